// et_static.cu -- et_T_static: Eq. 2 for callers that cannot allocate (code under CUDA graph capture,
// tight serving loops, harnesses that forbid cudaMalloc).  A variant of the all-pairs kernel k_pairs_T whose whole
// scratch -- the bounding box, the pooled fp32 records and the per-CTA partial sums -- lives in ONE file-scope
// `static __device__` array of ET_STATIC_SCRATCH_BYTES (8 MiB; every GPU that loads libet.so holds it until exit).
// The entry point calls no cudaMalloc / cudaFree / cudaMallocHost, creates no stream or event and never synchronises:
// it enqueues five kernels on the caller's stream and returns; the result goes to a DEVICE et_result of the caller.
//
// In host code the array's name `g_scratch` is a host-side stand-in, not a device address: et_static_setup (once per
// device, with that device current) asks cudaGetSymbolAddress for the device address and the kernels get that pointer.
//
// Every call shares the array and finds the previous call's contents in it: k_st_init resets the bounding box and
// the non-finite flag, k_st_prep rewrites every record row up to npad (padding rows as zeros), every CTA of k_st_pairs
// writes all of its partial-sum slots.  Two calls that overlap on the GPU (different streams, or two host threads)
// race on the array: callers serialise them.
//
// Same arithmetic as et_T in its difference form: records u = (x - c) sqrt(log2 e / (2 sigma^2)) rounded to fp32 with
// c the centre of the bounding box of the fp32-rounded coordinates, psi_ij = 2^(-|u_i - u_j|^2) by one MUFU.EX2
// (psi_pair, et_device.cuh), fp32 partial sums over 256 j, fp64 beyond, fixed-order reductions.
#include <cmath>
#include <cstdio>

#include "../../include/et.h"
#include "et_device.cuh"

namespace et {
namespace st {

constexpr size_t kScratchBytes = ET_STATIC_SCRATCH_BYTES;
constexpr size_t kHdrBytes = 4096;        // Header below
constexpr int kMaxGrid = 1024;            // CTAs of k_st_pairs: partial sums [kMaxGrid][4] doubles
constexpr size_t kPartOff = kHdrBytes, kRecOff = 65536;
static_assert(kPartOff + kMaxGrid * 4 * sizeof(double) <= kRecOff, "partials fit below the records");
constexpr int kMaxDevices = 64;
constexpr int kRows = 4;                  // i rows per thread
constexpr int kTI = kThreads * kRows;     // rows per tile = kPad

static __device__ __align__(256) unsigned char g_scratch[kScratchBytes];

struct Header {
    uint32_t mm[16];  // mm[2k] = min, mm[2k + 1] = max of coordinate k as order-preserving keys of the fp32 values
    int flag;         // != 0: a NaN / Inf was seen
};

// device address of g_scratch per device, filled by et_static_setup
unsigned char *g_dev_ptr[kMaxDevices] = {nullptr};
int g_num_sms[kMaxDevices] = {0};
thread_local char g_err[256] = {0};

et_status fail(et_status st, const char *msg)
{
    snprintf(g_err, sizeof(g_err), "%s", msg);
    return st;
}

__device__ __forceinline__ uint32_t f2key(float f)
{
    const uint32_t b = __float_as_uint(f);
    return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}
__device__ __forceinline__ float key2f(uint32_t k) { return __uint_as_float((k & 0x80000000u) ? (k & 0x7fffffffu) : ~k); }

// ---- kernels ------------------------------------------------------------------------------------------------
// what must start clean in the shared array: the bounding box and the flag (the previous call's are still there)
__global__ void k_st_init(Header *h)
{
    if (threadIdx.x < 8) { h->mm[2 * threadIdx.x] = 0xffffffffu; h->mm[2 * threadIdx.x + 1] = 0u; }
    if (threadIdx.x == 0) h->flag = 0;
}

// bounding box of the fp32-rounded coordinates of both samples (integer atomics: order-independent), non-finite flag
template <typename TIn>
__global__ void __launch_bounds__(256) k_st_minmax(const TIn *__restrict__ x, long long n, const TIn *__restrict__ xbar, long long nbar,
                                                  int dim, Header *h)
{
    uint32_t lo[ET_MAX_DIM], hi[ET_MAX_DIM];
#pragma unroll
    for (int k = 0; k < ET_MAX_DIM; ++k) { lo[k] = 0xffffffffu; hi[k] = 0u; }
    bool bad = false;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n + nbar; i += (long long)gridDim.x * blockDim.x) {
        const TIn *p = i < n ? x + i * dim : xbar + (i - n) * dim;
#pragma unroll
        for (int k = 0; k < ET_MAX_DIM; ++k)
            if (k < dim) {
                const double v = (double)p[k];
                if (!isfinite(v)) bad = true;
                const uint32_t key = f2key((float)v);
                lo[k] = min(lo[k], key);
                hi[k] = max(hi[k], key);
            }
    }
#pragma unroll
    for (int k = 0; k < ET_MAX_DIM; ++k)
        if (k < dim) {
            uint32_t a = lo[k], b = hi[k];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                a = min(a, __shfl_xor_sync(0xffffffffu, a, o));
                b = max(b, __shfl_xor_sync(0xffffffffu, b, o));
            }
            if ((threadIdx.x & 31) == 0) {
                atomicMin(&h->mm[2 * k], a);
                atomicMax(&h->mm[2 * k + 1], b);
            }
        }
    if (bad) atomicOr(&h->flag, 1);
}

// pooled records: rows [0, npadx) sample X (n real rows), rows [npadx, npad) sample Xbar; F floats per row:
// u[0 .. dim), the weight (1 on real rows, 0 on padding), zeros.  EVERY row is written (the array keeps old contents).
template <typename TIn>
__global__ void __launch_bounds__(256) k_st_prep(const TIn *__restrict__ x, long long n, const TIn *__restrict__ xbar, long long nbar,
                                                long long npadx, long long npad, int dim, double scale, const Header *__restrict__ h,
                                                float *__restrict__ rec)
{
    const int F = rec_floats(dim);
    double centre[ET_MAX_DIM];
#pragma unroll
    for (int k = 0; k < ET_MAX_DIM; ++k) centre[k] = k < dim ? 0.5 * ((double)key2f(h->mm[2 * k]) + (double)key2f(h->mm[2 * k + 1])) : 0.0;
    for (long long row = blockIdx.x * (long long)blockDim.x + threadIdx.x; row < npad; row += (long long)gridDim.x * blockDim.x) {
        const TIn *p = nullptr;
        if (row < npadx) { if (row < n) p = x + row * dim; }
        else if (row - npadx < nbar) p = xbar + (row - npadx) * dim;
        float *o = rec + row * F;
        if (!p) {
            for (int k = 0; k < F; ++k) o[k] = 0.0f;
            continue;
        }
#pragma unroll
        for (int k = 0; k < ET_MAX_DIM; ++k)
            if (k < dim) o[k] = (float)(((double)p[k] - centre[k]) * scale);
        o[dim] = 1.0f;
        for (int k = dim + 1; k < F; ++k) o[k] = 0.0f;
    }
}

// The variant of k_pairs_T (et_kernels.cuh): block sums S_xx, S_xb, S_bb of w_i w_j psi_ij over the upper triangle of
// kTI-row tiles, unit = (I, J), I <= J, dealt to the persistent CTAs round-robin; 256 j records staged in shared
// memory per step, 4 i rows per thread in registers; fp32 per pair and per 256-j partial, fp64 beyond; per-CTA sums in a
// fixed order, so the result depends only on the grid size.  Records and partial sums are in the static array.
// Tiles below nTx hold sample X, the others Xbar: slot = cls(I) + cls(J) = 0 (xx), 1 (xb), 2 (bb).
template <int D>
__global__ void __launch_bounds__(kThreads) k_st_pairs(const float *__restrict__ rec, int nT, int nTx, long long nunits,
                                                      double *__restrict__ partials)
{
    constexpr int F = rec_floats(D), F4 = F / 4;
    __shared__ float4 sj[kTileJ * F4];
    __shared__ double s_sum[4];
    __shared__ double s_warp[kThreads / 32];
    const int tid = threadIdx.x;
    if (tid < 4) s_sum[tid] = 0.0;
    for (long long unit = blockIdx.x; unit < nunits; unit += gridDim.x) {
        int I, J;
        unit_to_pair(unit, nT, I, J);
        const int slot = (I >= nTx ? 1 : 0) + (J >= nTx ? 1 : 0);
        float ui[kRows][D], wi[kRows];
#pragma unroll
        for (int r = 0; r < kRows; ++r) {
            const float4 *p = reinterpret_cast<const float4 *>(rec + ((long long)I * kTI + r * kThreads + tid) * F);
            float v[F];
#pragma unroll
            for (int q = 0; q < F4; ++q) {
                const float4 t = p[q];
                v[4 * q] = t.x; v[4 * q + 1] = t.y; v[4 * q + 2] = t.z; v[4 * q + 3] = t.w;
            }
#pragma unroll
            for (int k = 0; k < D; ++k) ui[r][k] = v[k];
            wi[r] = v[D];
        }
        double racc[kRows];
#pragma unroll
        for (int r = 0; r < kRows; ++r) racc[r] = 0.0;
        for (int sub = 0; sub < kTI / kTileJ; ++sub) {
            __syncthreads();
            {
                const float4 *p = reinterpret_cast<const float4 *>(rec + ((long long)J * kTI + sub * kTileJ + tid) * F);
#pragma unroll
                for (int q = 0; q < F4; ++q) sj[tid * F4 + q] = p[q];
            }
            __syncthreads();
            float acc[kRows];
#pragma unroll
            for (int r = 0; r < kRows; ++r) acc[r] = 0.f;
#pragma unroll 4
            for (int j = 0; j < kTileJ; ++j) {
                float uj[F];
#pragma unroll
                for (int q = 0; q < F4; ++q) {
                    const float4 t = sj[j * F4 + q];
                    uj[4 * q] = t.x; uj[4 * q + 1] = t.y; uj[4 * q + 2] = t.z; uj[4 * q + 3] = t.w;
                }
#pragma unroll
                for (int r = 0; r < kRows; ++r) acc[r] = __fmaf_rn(psi_pair<D>(ui[r], uj), uj[D], acc[r]);
            }
#pragma unroll
            for (int r = 0; r < kRows; ++r) racc[r] += (double)acc[r];
        }
        // the diagonal tile counted every ordered pair and psi_ii = 2^(-0) = 1 once per row
        const bool diag = I == J;
        double t = 0.0;
#pragma unroll
        for (int r = 0; r < kRows; ++r) t += (double)wi[r] * (diag ? racc[r] - (double)wi[r] : racc[r]);
        if (diag) t *= 0.5;
        t = warp_sum(t);
        if ((tid & 31) == 0) s_warp[tid >> 5] = t;
        __syncthreads();
        if (tid == 0) {
            double s = 0.0;
#pragma unroll
            for (int w = 0; w < kThreads / 32; ++w) s += s_warp[w];
            s_sum[slot] += s;
        }
    }
    __syncthreads();
    if (tid < 4) partials[(long long)blockIdx.x * 4 + tid] = s_sum[tid];
}

// Eq. 2 from the partial sums (CTAs in order) into the caller's DEVICE et_result; NaN terms if the inputs were not finite
__global__ void k_st_finish(const double *__restrict__ partials, int grid, long long n, long long nbar, const Header *__restrict__ h,
                            et_result *out)
{
    if (threadIdx.x || blockIdx.x) return;
    double S[3] = {0.0, 0.0, 0.0};
    for (int b = 0; b < grid; ++b)
        for (int s = 0; s < 3; ++s) S[s] += partials[(long long)b * 4 + s];
    et_result r;
    const double W = (double)n, Wb = (double)nbar;
    r.S_xx = S[0]; r.S_xb = S[1]; r.S_bb = S[2];
    r.W = W; r.Wbar = Wb;
    r.n_pairs = n * (n - 1) / 2 + nbar * (nbar - 1) / 2 + n * nbar;
    r.T_xx = r.S_xx / (W * (W - 1.0));
    r.T_bb = r.S_bb / (Wb * (Wb - 1.0));
    r.T_xb = r.S_xb / (W * Wb);
    r.T = r.T_xx + r.T_bb - r.T_xb;
    if (h->flag) r.T = r.T_xx = r.T_bb = r.T_xb = r.S_xx = r.S_bb = r.S_xb = nan("");
    *out = r;
}

}  // namespace st
}  // namespace et

using namespace et;

extern "C" {

const char *et_static_last_error(void) { return st::g_err; }

// Set-up, once per device: the device address of the static array (cudaGetSymbolAddress with that device current).
et_status et_static_setup(int device)
{
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return st::fail(ET_ERR_CUDA, "no CUDA device (there is no CPU fallback)");
    if (device < 0 || device >= ndev || device >= st::kMaxDevices) return st::fail(ET_ERR_INVALID, "et_static_setup: bad device index");
    if (st::g_dev_ptr[device]) return ET_OK;
    int prev = 0;
    if (cudaGetDevice(&prev) != cudaSuccess) return st::fail(ET_ERR_CUDA, "cudaGetDevice failed");
    if (cudaSetDevice(device) != cudaSuccess) return st::fail(ET_ERR_CUDA, "cudaSetDevice failed");
    unsigned char *ptr = nullptr;
    int sms = 0;
    const cudaError_t e1 = cudaGetSymbolAddress((void **)&ptr, st::g_scratch);
    const cudaError_t e2 = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
    cudaSetDevice(prev);
    if (e1 != cudaSuccess || !ptr) {
        snprintf(st::g_err, sizeof(st::g_err), "cudaGetSymbolAddress(g_scratch): %s", cudaGetErrorString(e1));
        return ET_ERR_CUDA;
    }
    if (e2 != cudaSuccess || sms < 1) return st::fail(ET_ERR_CUDA, "cudaDeviceGetAttribute(multiprocessor count) failed");
    st::g_num_sms[device] = sms;
    st::g_dev_ptr[device] = ptr;
    return ET_OK;
}

#define ST_LAUNCH_CHECK(what)                                                                        \
    do {                                                                                             \
        const cudaError_t e_ = cudaGetLastError();                                                   \
        if (e_ != cudaSuccess) {                                                                     \
            snprintf(st::g_err, sizeof(st::g_err), "et_T_static: %s: %s", what, cudaGetErrorString(e_)); \
            return ET_ERR_CUDA;                                                                      \
        }                                                                                            \
    } while (0)

et_status et_T_static(int device, void *cuda_stream, const void *x, int64_t n, const void *xbar, int64_t nbar, int dim, et_dtype dtype,
                      double sigma, et_result *out_device)
{
    if (!x || !xbar || !out_device) return st::fail(ET_ERR_INVALID, "et_T_static: null pointer");
    if (n < 2 || nbar < 2) return st::fail(ET_ERR_INVALID, "et_T_static: n and nbar must be >= 2 (Eq. 2 divides by n(n-1))");
    if (dim < 1 || dim > ET_MAX_DIM) return st::fail(ET_ERR_INVALID, "et_T_static: dim out of range");
    if (dtype != ET_F32 && dtype != ET_F64) return st::fail(ET_ERR_INVALID, "et_T_static: bad dtype");
    if (!(sigma > 0.0) || !std::isfinite(sigma)) return st::fail(ET_ERR_SIGMA, "et_T_static: sigma must be finite and > 0");
    if (device < 0 || device >= st::kMaxDevices || !st::g_dev_ptr[device])
        return st::fail(ET_ERR_INVALID, "et_T_static: call et_static_setup(device) first (outside graph capture)");
    const int F = rec_floats(dim);
    const long long npadx = (n + kPad - 1) / kPad * kPad, npad = npadx + (nbar + kPad - 1) / kPad * kPad;
    const unsigned long long need = st::kRecOff + (unsigned long long)npad * F * sizeof(float);
    if (n > (1ll << 30) || nbar > (1ll << 30) || need > st::kScratchBytes) {
        snprintf(st::g_err, sizeof(st::g_err),
                 "et_T_static: %lld padded rows x %d bytes need %llu bytes of scratch, the static array holds %llu "
                 "(ET_STATIC_SCRATCH_BYTES): use et_T for samples of this size",
                 npad, F * 4, need, (unsigned long long)st::kScratchBytes);
        return ET_ERR_INVALID;
    }
    int cur = -1;
    if (cudaGetDevice(&cur) != cudaSuccess) return st::fail(ET_ERR_CUDA, "cudaGetDevice failed");
    if (cur != device && cudaSetDevice(device) != cudaSuccess) return st::fail(ET_ERR_CUDA, "cudaSetDevice failed");
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    unsigned char *base = st::g_dev_ptr[device];
    st::Header *hdr = reinterpret_cast<st::Header *>(base);
    double *partials = reinterpret_cast<double *>(base + st::kPartOff);
    float *rec = reinterpret_cast<float *>(base + st::kRecOff);
    const int sms = st::g_num_sms[device];
    const double scale = std::sqrt(1.4426950408889634074 / (2.0 * sigma * sigma));

    st::k_st_init<<<1, 32, 0, s>>>(hdr);
    ST_LAUNCH_CHECK("k_st_init");
    if (dtype == ET_F32) {
        st::k_st_minmax<float><<<sms * 4, 256, 0, s>>>(static_cast<const float *>(x), n, static_cast<const float *>(xbar), nbar, dim, hdr);
        ST_LAUNCH_CHECK("k_st_minmax");
        st::k_st_prep<float><<<sms * 4, 256, 0, s>>>(static_cast<const float *>(x), n, static_cast<const float *>(xbar), nbar, npadx, npad, dim, scale, hdr, rec);
    } else {
        st::k_st_minmax<double><<<sms * 4, 256, 0, s>>>(static_cast<const double *>(x), n, static_cast<const double *>(xbar), nbar, dim, hdr);
        ST_LAUNCH_CHECK("k_st_minmax");
        st::k_st_prep<double><<<sms * 4, 256, 0, s>>>(static_cast<const double *>(x), n, static_cast<const double *>(xbar), nbar, npadx, npad, dim, scale, hdr, rec);
    }
    ST_LAUNCH_CHECK("k_st_prep");
    const int nT = (int)(npad / st::kTI), nTx = (int)(npadx / st::kTI);
    const long long nunits = (long long)nT * (nT + 1) / 2;
    int grid = 2 * sms < st::kMaxGrid ? 2 * sms : st::kMaxGrid;
    if ((long long)grid > nunits) grid = (int)nunits;
    switch (dim) {
        case 1: st::k_st_pairs<1><<<grid, kThreads, 0, s>>>(rec, nT, nTx, nunits, partials); break;
        case 2: st::k_st_pairs<2><<<grid, kThreads, 0, s>>>(rec, nT, nTx, nunits, partials); break;
        case 3: st::k_st_pairs<3><<<grid, kThreads, 0, s>>>(rec, nT, nTx, nunits, partials); break;
        case 4: st::k_st_pairs<4><<<grid, kThreads, 0, s>>>(rec, nT, nTx, nunits, partials); break;
        case 5: st::k_st_pairs<5><<<grid, kThreads, 0, s>>>(rec, nT, nTx, nunits, partials); break;
        case 6: st::k_st_pairs<6><<<grid, kThreads, 0, s>>>(rec, nT, nTx, nunits, partials); break;
        case 7: st::k_st_pairs<7><<<grid, kThreads, 0, s>>>(rec, nT, nTx, nunits, partials); break;
        default: st::k_st_pairs<8><<<grid, kThreads, 0, s>>>(rec, nT, nTx, nunits, partials); break;
    }
    ST_LAUNCH_CHECK("k_st_pairs");
    st::k_st_finish<<<1, 32, 0, s>>>(partials, grid, n, nbar, hdr, out_device);
    ST_LAUNCH_CHECK("k_st_finish");
    return ET_OK;
}

}  // extern "C"
