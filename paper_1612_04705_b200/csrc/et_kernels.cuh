// et_kernels.cuh -- the CUDA kernels of libet.so (sm_100a).
//
// Pooled layout ("records"): events are grouped by class (2 classes X / Xbar, or the 4 classes of the Sect. 5
// split), every class segment padded to a multiple of et::kPad rows.  Row r is rec_floats(dim) floats:
// u[0..dim) = (x - centre) * sqrt(log2(e) / (2 sigma^2)) rounded to fp32, then the weight w (1 when unweighted,
// 0 on padding rows), then zeros.  psi_ij = 2^(-|u_i - u_j|^2), padding contributes w = 0.
#pragma once
#include "et_device.cuh"

namespace et {

// ------------------------------------------------------------------------------------------------ prep
// Bounding box of the coordinates (for the centre) and the non-finite check.  mm[2*k] = min, mm[2*k+1] = max as
// order-preserving uint32 keys of the fp32-rounded values (mm[16], mm[17]: min / max of the fp32-rounded weights);
// flag[0] != 0 when a NaN/Inf was seen.
__device__ __forceinline__ uint32_t f2key(float f)
{
    uint32_t b = __float_as_uint(f);
    return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}
__host__ __device__ inline float key2f(uint32_t k)
{
    uint32_t b = (k & 0x80000000u) ? (k & 0x7fffffffu) : ~k;
#ifdef __CUDA_ARCH__
    return __uint_as_float(b);
#else
    float f;
    memcpy(&f, &b, 4);
    return f;
#endif
}

template <typename TIn>
__global__ void k_minmax(const TIn *__restrict__ x, long long n, int dim, const double *__restrict__ w,
                         uint32_t *__restrict__ mm, int *__restrict__ flag)
{
    uint32_t lo[8], hi[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) { lo[k] = 0xffffffffu; hi[k] = 0u; }
    bool bad = false;
    uint32_t wlo = 0xffffffffu, whi = 0u;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
#pragma unroll
        for (int k = 0; k < 8; ++k)
            if (k < dim) {
                const double v = (double)x[i * dim + k];
                if (!isfinite(v)) bad = true;
                const uint32_t key = f2key((float)v);
                lo[k] = min(lo[k], key);
                hi[k] = max(hi[k], key);
            }
        if (w) {
            if (!isfinite(w[i])) bad = true;
            const uint32_t key = f2key((float)w[i]);
            wlo = min(wlo, key);
            whi = max(whi, key);
        }
    }
    if (w) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            wlo = min(wlo, __shfl_xor_sync(0xffffffffu, wlo, o));
            whi = max(whi, __shfl_xor_sync(0xffffffffu, whi, o));
        }
        if ((threadIdx.x & 31) == 0) {
            atomicMin(&mm[16], wlo);
            atomicMax(&mm[17], whi);
        }
    }
#pragma unroll
    for (int k = 0; k < 8; ++k)
        if (k < dim) {
            uint32_t a = lo[k], b = hi[k];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                a = min(a, __shfl_xor_sync(0xffffffffu, a, o));
                b = max(b, __shfl_xor_sync(0xffffffffu, b, o));
            }
            if ((threadIdx.x & 31) == 0) {
                atomicMin(&mm[2 * k], a);
                atomicMax(&mm[2 * k + 1], b);
            }
        }
    if (bad) atomicOr(flag, 1);
}

struct PrepParams {
    double centre[8];
    double scale;        // sqrt(log2(e) / (2 sigma^2))
    long long n, nbar;   // sizes of the two source arrays
    long long npad;      // rows of the pooled layout
    int dim;
    int ncls;
    long long seg_pos[kMaxCls + 1];    // first padded row of each class segment (seg_pos[ncls] = npad)
    long long seg_count[kMaxCls];      // real rows in each class segment
    // Morton key of every row for the row order of the tensor-core contraction (et_tc.cuh): class << 20 | the interleaved top
    // key_bits bits per axis of (x - centre) / half range, in fp64 from the INPUT coordinates, so the key does not depend on
    // sigma (a sigma scan and its single calls order the rows alike); padding rows get the largest key of their class
    double inv_half[8];                // 1 / half range of coordinate k over the bounding box (0: a degenerate axis)
    int key_bits;
    uint32_t *key;                     // [npad], or nullptr
};

// Writes the pooled records.  src == nullptr: two classes, class 0 = x in input order, class 1 = xbar.
// src != nullptr: src[row] is the pooled source index (0..n-1 -> x, n.. -> xbar) of a real row, -1 on padding.
template <typename TIn>
__global__ void k_prep(const TIn *__restrict__ x, const TIn *__restrict__ xbar, const double *__restrict__ wx,
                       const double *__restrict__ wxbar, const int *__restrict__ src, PrepParams P,
                       float *__restrict__ rec)
{
    const int F = rec_floats(P.dim);
    for (long long row = blockIdx.x * (long long)blockDim.x + threadIdx.x; row < P.npad;
         row += (long long)gridDim.x * blockDim.x) {
        long long s = -1;
        if (src) {
            s = src[row];
        } else {
            if (row < P.seg_pos[1]) { if (row < P.n) s = row; }
            else if (row - P.seg_pos[1] < P.nbar) s = P.n + (row - P.seg_pos[1]);
        }
        float *o = rec + row * F;
        int cls = 0;
        for (int c = 1; c < P.ncls; ++c)
            if (row >= P.seg_pos[c]) cls = c;
        if (s < 0) {
            for (int k = 0; k < F; ++k) o[k] = 0.0f;
            if (P.key) P.key[row] = ((uint32_t)cls << 20) | 0x000fffffu;
            continue;
        }
        const TIn *p = s < P.n ? x + s * P.dim : xbar + (s - P.n) * P.dim;
        for (int k = 0; k < P.dim; ++k) o[k] = (float)(((double)p[k] - P.centre[k]) * P.scale);
        if (P.key) {
            const int top = (1 << P.key_bits) - 1;
            uint32_t q[8], m = 0u;
            for (int k = 0; k < P.dim; ++k) {
                const double t = (((double)p[k] - P.centre[k]) * P.inv_half[k] + 1.0) * 0.5 * (double)(1 << P.key_bits);
                q[k] = (uint32_t)min(max((int)t, 0), top);
            }
            for (int b = P.key_bits - 1; b >= 0; --b)
                for (int k = 0; k < P.dim; ++k) m = (m << 1) | ((q[k] >> b) & 1u);
            P.key[row] = ((uint32_t)cls << 20) | m;
        }
        double w = 1.0;
        if (wx) w = s < P.n ? wx[s] : wxbar[s - P.n];
        o[P.dim] = (float)w;
        for (int k = P.dim + 1; k < F; ++k) o[k] = 0.0f;
    }
}

// ------------------------------------------------------------------------------------------------ all pairs
// w_j psi_ij rounded to the nearest multiple of the grid step G that `magic` = 1.5 * 2^23 G encodes (magic = 0: no
// rounding).  The CUDA-core permutation kernels sum these terms: up to kFlushJ of them, |term| <= 2^23 G / kFlushJ, add up
// EXACTLY in fp32, so Q_p, the row sums r_i and S are sums of the same numbers whatever the labels (kFlushJ, et_device.cuh).
__device__ __forceinline__ float grid_term(float psi, float w, float magic) { return __fadd_rn(__fmaf_rn(psi, w, magic), -magic); }

// One j record from shared memory: coordinates and weight.
template <int D>
struct JRec {
    float u[D];
    float w;
};
template <int D>
__device__ __forceinline__ JRec<D> load_jrec(const float4 *__restrict__ sj, int j)
{
    constexpr int F4 = rec_floats(D) / 4;
    float v[F4 * 4];
#pragma unroll
    for (int q = 0; q < F4; ++q) {
        const float4 t = sj[j * F4 + q];
        v[4 * q] = t.x; v[4 * q + 1] = t.y; v[4 * q + 2] = t.z; v[4 * q + 3] = t.w;
    }
    JRec<D> r;
#pragma unroll
    for (int k = 0; k < D; ++k) r.u[k] = v[k];
    r.w = v[D];
    return r;
}

// K-T: class-pair block sums S[c1][c2] = sum over unordered pairs of w_i w_j psi_ij (Eq. 2's three sums, or the ten
// of the four-class split), over the upper triangle of i-tiles.  Work unit = (I, J), I <= J, tiles of 256*R rows;
// fp32 per pair and per 128-j partial row sum, fp64 from there on; per-unit block reduction in a fixed order, so the
// result depends only on the grid size.
// Packed FP32 pipe, two j per instruction: the j records are staged in shared memory as PAIRS, float2 k of pair p =
// (-u_{2p,k}, -u_{2p+1,k}), float2 D = (w_2p, w_2p+1), and every thread's R i rows enter as (u_ik, u_ik) -- ONE register: ptxas encodes the pair as the scalar-broadcast operand form R.F32 of FADD2 / FFMA2 (round 2: a materialised register pair per coordinate cost 20 registers at D = 5: Gram form 128 -> 80 registers, 3 CTAs per SM instead of 2, config 4 578 -> 561 ms) -- so that one FADD2 / FFMA2 does the
// subtraction / square-accumulate of (i, 2p) and (i, 2p+1) at once.  Each half of a packed instruction rounds like the
// scalar one (u_i + (-u_j) == u_i - u_j exactly), so psi is bit-identical to psi_pair<D>.  The packed instructions
// halve the issue slots per pair (2D+1 FP32 lane-ops and one MUFU.EX2 per pair stay): measured 2.3 -> 2.8e12 pairs/s
// at D = 5 (profiles/r01_pipe_probes.md).
// skip_mask: bit c1 * 4 + c2 (c1 <= c2) set = tile pairs of that class pair are not evaluated (their slot stays 0);
// the guard-band escalation needs six of the ten class-pair sums only.  Units unit0 + k * unit_step (k = 0, 1, ...) are
// this launch's share: (0, 1) on one GPU, (rank, world) when the unit range is sharded over ranks.
// GRAM: e_ij = |u_i|^2 + |u_j|^2 + sum_k u_ik (-2 u_jk), and the row's constant is taken out of the exponent:
// psi_ij = 2^(-|u_i|^2) 2^(-e'_ij), e'_ij = |u_j|^2 + sum_k u_ik (-2 u_jk) -- D FFMA2 per two pairs instead of D FADD2, one
// FMUL2 and D - 1 FFMA2, i.e. D + 1 instead of 2 D + 1 FP32-pipe lane-ops per pair with the accumulation (D = 5: 6 instead
// of 11; the kernel is then bound by the 16 MUFU.EX2 per clock and SM); the factor 2^(-|u_i|^2) multiplies the row's fp32
// partial sum once per 256 j, in double.  2^(-e') <= 2^(|u_i|^2) <= 2^umax2: the host keeps umax2 <= 96 for this form.  Every operation rounds a value of size <= 2 (|u_i|^2 + |u_j|^2)
// instead of the small difference, so psi carries a relative error of about kGramErr umax2 (umax2 = the largest |u|^2: the
// squared half diagonal of the bounding box in units of sigma sqrt(2 / log2 e)) -- zero-mean rounding noise that averages
// over the pairs, plus a per-event part from the rounding of |u_i|^2 that acts like a weight 1 + O(1e-7 umax2) on event i.
// The host takes this form only for samples large enough for the noise to average far below the 1e-6 tolerance of T and
// compact enough in units of sigma (run_pairs_T); the guard band of the escalation carries the extra term.
constexpr double kGramErr = 8.262958e-08;  // 2^-23 ln 2
template <int D, int R, bool GRAM>
__global__ void __launch_bounds__(kThreads) k_pairs_T(const float *__restrict__ rec, int nT,
                                                     const uint8_t *__restrict__ tile_cls, long long nunits,
                                                     unsigned skip_mask, int unit0, int unit_step,
                                                     double *__restrict__ partials)
{
    constexpr int F = rec_floats(D), F4 = F / 4, TI = kThreads * R;
    constexpr int NP = D + (GRAM ? 2 : 1), NLD = (NP + 1) / 2;  // float2 entries / LDS.128 per j pair
    constexpr int WI = GRAM ? D + 1 : D;                        // entry that holds the weights
    __shared__ float4 sj[kTileJ / 2 * NLD];
    __shared__ double s_sum[kSumSlots];
    __shared__ double s_warp[kThreads / 32];
    const int tid = threadIdx.x;
    if (tid < kSumSlots) s_sum[tid] = 0.0;

    for (long long unit = unit0 + (long long)unit_step * blockIdx.x; unit < nunits; unit += (long long)unit_step * gridDim.x) {
        int I, J;
        unit_to_pair(unit, nT, I, J);
        const int slot = tile_cls[(long long)I * TI / kPad] * 4 + tile_cls[(long long)J * TI / kPad];
        if (skip_mask >> slot & 1u) continue;
        float2 ui[R][D];
        double rs[R];           // GRAM: 2^(-|u_i|^2), the factor of the row taken out of the exponent; else 1
        float wi[R], self[R];   // self: w_i psi_ii / rs as this kernel evaluates it (w_i exactly with the difference form)
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const float4 *p = reinterpret_cast<const float4 *>(rec + ((long long)I * TI + r * kThreads + tid) * F);
            float v[F];
#pragma unroll
            for (int q = 0; q < F4; ++q) {
                const float4 t = __ldg(p + q);
                v[4 * q] = t.x; v[4 * q + 1] = t.y; v[4 * q + 2] = t.z; v[4 * q + 3] = t.w;
            }
            // (u_ik, u_ik) from one register: the packed instructions take it as a scalar-broadcast operand (R.F32)
#pragma unroll
            for (int k = 0; k < D; ++k) ui[r][k] = make_float2(v[k], v[k]);
            wi[r] = v[D];
            self[r] = v[D];
            rs[r] = 1.0;
            if (GRAM) {
                float na = __fmul_rn(v[0], v[0]);
#pragma unroll
                for (int k = 1; k < D; ++k) na = __fmaf_rn(v[k], v[k], na);
                rs[r] = exp2(-(double)na);
                // 2^(-e'_ii) by the instruction sequence of the loop below (each half of a packed instruction rounds
                // like the scalar one): what the diagonal tile adds for j = i, removed again after the loop
                float e = na;
#pragma unroll
                for (int k = 0; k < D; ++k) e = __fmaf_rn(v[k], -2.f * v[k], e);
                self[r] = __fmul_rn(ex2_approx(-e), v[D]);
            }
        }
        double racc[R];
#pragma unroll
        for (int r = 0; r < R; ++r) racc[r] = 0.0;

        for (int sub = 0; sub < TI / kTileJ; ++sub) {
            __syncthreads();
            {
                const float4 *p = reinterpret_cast<const float4 *>(rec + ((long long)J * TI + sub * kTileJ + tid) * F);
                float v[F];
#pragma unroll
                for (int q = 0; q < F4; ++q) {
                    const float4 t = __ldg(p + q);
                    v[4 * q] = t.x; v[4 * q + 1] = t.y; v[4 * q + 2] = t.z; v[4 * q + 3] = t.w;
                }
                float *o = reinterpret_cast<float *>(sj) + (tid >> 1) * (NLD * 4) + (tid & 1);
                if (GRAM) {
                    float nb = __fmul_rn(v[0], v[0]);
#pragma unroll
                    for (int k = 1; k < D; ++k) nb = __fmaf_rn(v[k], v[k], nb);
#pragma unroll
                    for (int k = 0; k < D; ++k) o[2 * k] = -2.f * v[k];
                    o[2 * D] = nb;
                } else {
#pragma unroll
                    for (int k = 0; k < D; ++k) o[2 * k] = -v[k];
                }
                o[2 * WI] = v[D];
                if (NP & 1) o[2 * NP] = 0.f;
            }
            __syncthreads();
            float2 acc[R];
#pragma unroll
            for (int r = 0; r < R; ++r) acc[r] = make_float2(0.f, 0.f);
#pragma unroll 4
            for (int jp = 0; jp < kTileJ / 2; ++jp) {
                float2 nu[2 * NLD];
#pragma unroll
                for (int q = 0; q < NLD; ++q) {
                    const float4 t = sj[jp * NLD + q];
                    nu[2 * q] = make_float2(t.x, t.y);
                    nu[2 * q + 1] = make_float2(t.z, t.w);
                }
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    float2 e;
                    if (GRAM) {
                        e = nu[D];
#pragma unroll
                        for (int k = 0; k < D; ++k) e = __ffma2_rn(ui[r][k], nu[k], e);
                    } else {
                        float2 d = __fadd2_rn(ui[r][0], nu[0]);
                        e = __fmul2_rn(d, d);
#pragma unroll
                        for (int k = 1; k < D; ++k) {
                            d = __fadd2_rn(ui[r][k], nu[k]);
                            e = __ffma2_rn(d, d, e);
                        }
                    }
                    acc[r] = __ffma2_rn(make_float2(ex2_approx(-e.x), ex2_approx(-e.y)), nu[WI], acc[r]);
                }
            }
#pragma unroll
            for (int r = 0; r < R; ++r) racc[r] += (double)acc[r].x + (double)acc[r].y;
        }
        double t = 0.0;
        const bool diag = I == J;
#pragma unroll
        for (int r = 0; r < R; ++r) t += (double)wi[r] * rs[r] * (diag ? racc[r] - (double)self[r] : racc[r]);
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
    if (tid < kSumSlots) partials[(long long)blockIdx.x * kSumSlots + tid] = s_sum[tid];
}

// K-T for several sigma at once (the sigma scan of PAPER.md:73-81): the records are scaled for
// sigma_0, e = |u_i - u_j|^2 is evaluated once per pair and psi_s = 2^(-e rho_s), rho_s = (sigma_0 / sigma_s)^2, costs
// one FMUL2, two MUFU.EX2 and one FFMA2 per extra sigma and pair of j instead of the 2D packed distance instructions.
// Same tiling, precision rules and reduction order as k_pairs_T; partials[block][s][slot].
template <int D, int R, int NS>
__global__ void __launch_bounds__(kThreads) k_pairs_T_multi(const float *__restrict__ rec, int nT,
                                                           const uint8_t *__restrict__ tile_cls, long long nunits,
                                                           const float *__restrict__ rho, double *__restrict__ partials)
{
    constexpr int F = rec_floats(D), F4 = F / 4, TI = kThreads * R;
    constexpr int NP = D + 1, NLD = (NP + 1) / 2;
    __shared__ float4 sj[kTileJ / 2 * NLD];
    __shared__ double s_sum[NS][kSumSlots];
    __shared__ double s_warp[NS][kThreads / 32];
    const int tid = threadIdx.x;
    for (int k = tid; k < NS * kSumSlots; k += kThreads) s_sum[k / kSumSlots][k % kSumSlots] = 0.0;
    float2 nrho[NS];  // -rho_s duplicated (nrho[0] unused: rho_0 = 1)
#pragma unroll
    for (int s = 0; s < NS; ++s) nrho[s] = make_float2(-rho[s], -rho[s]);

    for (long long unit = blockIdx.x; unit < nunits; unit += gridDim.x) {
        int I, J;
        unit_to_pair(unit, nT, I, J);
        float2 ui[R][D];
        float wi[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const float4 *p = reinterpret_cast<const float4 *>(rec + ((long long)I * TI + r * kThreads + tid) * F);
            float v[F];
#pragma unroll
            for (int q = 0; q < F4; ++q) {
                const float4 t = __ldg(p + q);
                v[4 * q] = t.x; v[4 * q + 1] = t.y; v[4 * q + 2] = t.z; v[4 * q + 3] = t.w;
            }
#pragma unroll
            for (int k = 0; k < D; ++k) ui[r][k] = make_float2(v[k], v[k]);
            wi[r] = v[D];
        }
        double racc[NS][R];
#pragma unroll
        for (int s = 0; s < NS; ++s)
#pragma unroll
            for (int r = 0; r < R; ++r) racc[s][r] = 0.0;

        for (int sub = 0; sub < TI / kTileJ; ++sub) {
            __syncthreads();
            {
                const float4 *p = reinterpret_cast<const float4 *>(rec + ((long long)J * TI + sub * kTileJ + tid) * F);
                float v[F];
#pragma unroll
                for (int q = 0; q < F4; ++q) {
                    const float4 t = __ldg(p + q);
                    v[4 * q] = t.x; v[4 * q + 1] = t.y; v[4 * q + 2] = t.z; v[4 * q + 3] = t.w;
                }
                float *o = reinterpret_cast<float *>(sj) + (tid >> 1) * (NLD * 4) + (tid & 1);
#pragma unroll
                for (int k = 0; k < D; ++k) o[2 * k] = -v[k];
                o[2 * D] = v[D];
                if (NP & 1) o[2 * NP] = 0.f;
            }
            __syncthreads();
            float2 acc[NS][R];
#pragma unroll
            for (int s = 0; s < NS; ++s)
#pragma unroll
                for (int r = 0; r < R; ++r) acc[s][r] = make_float2(0.f, 0.f);
#pragma unroll 2
            for (int jp = 0; jp < kTileJ / 2; ++jp) {
                float2 nu[2 * NLD];
#pragma unroll
                for (int q = 0; q < NLD; ++q) {
                    const float4 t = sj[jp * NLD + q];
                    nu[2 * q] = make_float2(t.x, t.y);
                    nu[2 * q + 1] = make_float2(t.z, t.w);
                }
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    float2 d = __fadd2_rn(ui[r][0], nu[0]);
                    float2 e = __fmul2_rn(d, d);
#pragma unroll
                    for (int k = 1; k < D; ++k) {
                        d = __fadd2_rn(ui[r][k], nu[k]);
                        e = __ffma2_rn(d, d, e);
                    }
                    acc[0][r] = __ffma2_rn(make_float2(ex2_approx(-e.x), ex2_approx(-e.y)), nu[D], acc[0][r]);
#pragma unroll
                    for (int s = 1; s < NS; ++s) {
                        const float2 es = __fmul2_rn(e, nrho[s]);
                        acc[s][r] = __ffma2_rn(make_float2(ex2_approx(es.x), ex2_approx(es.y)), nu[D], acc[s][r]);
                    }
                }
            }
#pragma unroll
            for (int s = 0; s < NS; ++s)
#pragma unroll
                for (int r = 0; r < R; ++r) racc[s][r] += (double)acc[s][r].x + (double)acc[s][r].y;
        }
        const bool diag = I == J;
#pragma unroll
        for (int s = 0; s < NS; ++s) {
            double t = 0.0;
#pragma unroll
            for (int r = 0; r < R; ++r) t += (double)wi[r] * (diag ? racc[s][r] - (double)wi[r] : racc[s][r]);
            if (diag) t *= 0.5;
            t = warp_sum(t);
            if ((tid & 31) == 0) s_warp[s][tid >> 5] = t;
        }
        __syncthreads();
        if (tid < NS) {
            double sum = 0.0;
#pragma unroll
            for (int w = 0; w < kThreads / 32; ++w) sum += s_warp[tid][w];
            s_sum[tid][tile_cls[(long long)I * TI / kPad] * 4 + tile_cls[(long long)J * TI / kPad]] += sum;
        }
    }
    __syncthreads();
    for (int k = tid; k < NS * kSumSlots; k += kThreads) partials[(long long)blockIdx.x * NS * kSumSlots + k] = s_sum[k / kSumSlots][k % kSumSlots];
}

// K-ROW: full row sums by class of j, rowsum[c][i] = sum_{j in class c, j != i} w_j psi_ij, for every pooled row.
// Work unit = one i-tile of 256*R rows against all j; units handed out by an atomic counter (each row is summed by
// one CTA in a fixed j order, so the result does not depend on the schedule).
struct RowSegs {
    int jt_begin[kMaxCls + 1];  // j sub-tile (kTileJ rows) range of each class segment
};
template <int D, int R, int C>
__global__ void __launch_bounds__(kThreads) k_pairs_rows(const float *__restrict__ rec, int nT, long long npad,
                                                        const uint8_t *__restrict__ tile_cls, RowSegs segs, float magic,
                                                        int *__restrict__ counter, double *__restrict__ rowsum)
{
    constexpr int F = rec_floats(D), F4 = F / 4, TI = kThreads * R;
    __shared__ float4 sj[kTileJ * F4];
    __shared__ int s_unit;
    const int tid = threadIdx.x;
    for (;;) {
        __syncthreads();
        if (tid == 0) s_unit = atomicAdd(counter, 1);
        __syncthreads();
        const int I = s_unit;
        if (I >= nT) break;
        float ui[R][D], wi[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const float4 *p = reinterpret_cast<const float4 *>(rec + ((long long)I * TI + r * kThreads + tid) * F);
            float v[F];
#pragma unroll
            for (int q = 0; q < F4; ++q) {
                const float4 t = __ldg(p + q);
                v[4 * q] = t.x; v[4 * q + 1] = t.y; v[4 * q + 2] = t.z; v[4 * q + 3] = t.w;
            }
#pragma unroll
            for (int k = 0; k < D; ++k) ui[r][k] = v[k];
            wi[r] = v[D];
        }
        const int ci = tile_cls[(long long)I * TI / kPad];
        double racc[R][C];
#pragma unroll
        for (int c = 0; c < C; ++c) {
#pragma unroll
            for (int r = 0; r < R; ++r) racc[r][c] = 0.0;
            for (int jt = segs.jt_begin[c]; jt < segs.jt_begin[c + 1]; ++jt) {
                __syncthreads();
                {
                    const float4 *p = reinterpret_cast<const float4 *>(rec + ((long long)jt * kTileJ + tid) * F);
#pragma unroll
                    for (int q = 0; q < F4; ++q) sj[tid * F4 + q] = __ldg(p + q);
                }
                __syncthreads();
                // fp32 over kFlushJ pairs only (see kFlushJ), fp64 beyond
                for (int jb = 0; jb < kTileJ; jb += kFlushJ) {
                    float acc[R];
#pragma unroll
                    for (int r = 0; r < R; ++r) acc[r] = 0.0f;
#pragma unroll 4
                    for (int j = jb; j < jb + kFlushJ; ++j) {
                        const JRec<D> rj = load_jrec<D>(sj, j);
#pragma unroll
                        for (int r = 0; r < R; ++r) acc[r] = __fadd_rn(acc[r], grid_term(psi_pair<D>(ui[r], rj.u), rj.w, magic));
                    }
#pragma unroll
                    for (int r = 0; r < R; ++r) racc[r][c] += (double)acc[r];
                }
            }
            // the row's own term w_i * psi_ii = w_i sits in its own class
            if (c == ci) {
#pragma unroll
                for (int r = 0; r < R; ++r) racc[r][c] -= (double)grid_term(1.0f, wi[r], magic);
            }
#pragma unroll
            for (int r = 0; r < R; ++r) rowsum[(long long)c * npad + (long long)I * TI + r * kThreads + tid] = racc[r][c];
        }
    }
}

// K-PERM (CUDA cores): Q_c = sum_{i<j} a_ic a_jc w_i w_j psi_ij for the 32 label columns of one mask word, each psi
// evaluated once and fanned out to 32 fp32 accumulators per row (y_ic = sum_j w_j a_jc psi_ij), over the upper
// triangle of 512-row tiles.  fp32 over 256 j, then fp64 per thread across all its units; one block reduction at
// the end.  Columns: c = 0 is the observed labelling, c = p + 1 permutation p.
template <int D>
__global__ void __launch_bounds__(kThreads, 1) k_perm32(const float *__restrict__ rec, const uint32_t *__restrict__ maskg,
                                                       int nT, long long nunits, float magic, double *__restrict__ partialQ)
{
    constexpr int R = 2, F = rec_floats(D), F4 = F / 4, TI = kThreads * R;
    __shared__ float4 sj[kTileJ * F4];
    __shared__ float4 lab[kTileJ * 8];  // lab[j][c] = a_jc as 0.f / 1.f
    const int tid = threadIdx.x;
    double q[32];
#pragma unroll
    for (int c = 0; c < 32; ++c) q[c] = 0.0;

    for (long long unit = blockIdx.x; unit < nunits; unit += gridDim.x) {
        int I, J;
        unit_to_pair(unit, nT, I, J);
        float ui[R][D], wi[R];
        uint32_t mi[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const long long row = (long long)I * TI + r * kThreads + tid;
            const float4 *p = reinterpret_cast<const float4 *>(rec + row * F);
            float v[F];
#pragma unroll
            for (int qq = 0; qq < F4; ++qq) {
                const float4 t = __ldg(p + qq);
                v[4 * qq] = t.x; v[4 * qq + 1] = t.y; v[4 * qq + 2] = t.z; v[4 * qq + 3] = t.w;
            }
#pragma unroll
            for (int k = 0; k < D; ++k) ui[r][k] = v[k];
            wi[r] = v[D];
            mi[r] = __ldg(maskg + row);
        }
        const bool diag = I == J;
        const double f = diag ? 0.5 : 1.0;
        for (int sub = 0; sub < TI / kTileJ; ++sub) {
            __syncthreads();
            {
                const long long row = (long long)J * TI + sub * kTileJ + tid;
                const float4 *p = reinterpret_cast<const float4 *>(rec + row * F);
#pragma unroll
                for (int qq = 0; qq < F4; ++qq) sj[tid * F4 + qq] = __ldg(p + qq);
                const uint32_t m = __ldg(maskg + row);
#pragma unroll
                for (int c4 = 0; c4 < 8; ++c4) {
                    float4 l;
                    l.x = (m >> (4 * c4) & 1u) ? 1.f : 0.f;
                    l.y = (m >> (4 * c4 + 1) & 1u) ? 1.f : 0.f;
                    l.z = (m >> (4 * c4 + 2) & 1u) ? 1.f : 0.f;
                    l.w = (m >> (4 * c4 + 3) & 1u) ? 1.f : 0.f;
                    lab[tid * 8 + c4] = l;
                }
            }
            __syncthreads();
            // fp32 over kFlushJ pairs only (see kFlushJ), fp64 beyond
            for (int jb = 0; jb < kTileJ; jb += kFlushJ) {
                float y[R][32];
#pragma unroll
                for (int r = 0; r < R; ++r)
#pragma unroll
                    for (int c = 0; c < 32; ++c) y[r][c] = 0.f;
#pragma unroll 2
                for (int j = jb; j < jb + kFlushJ; ++j) {
                    const JRec<D> rj = load_jrec<D>(sj, j);
                    float ps[R];
#pragma unroll
                    for (int r = 0; r < R; ++r) ps[r] = grid_term(psi_pair<D>(ui[r], rj.u), rj.w, magic);  // w_j psi_ij on the grid
#pragma unroll
                    for (int c4 = 0; c4 < 8; ++c4) {
                        const float4 l = lab[j * 8 + c4];
#pragma unroll
                        for (int r = 0; r < R; ++r) {
                            y[r][4 * c4] = __fmaf_rn(ps[r], l.x, y[r][4 * c4]);
                            y[r][4 * c4 + 1] = __fmaf_rn(ps[r], l.y, y[r][4 * c4 + 1]);
                            y[r][4 * c4 + 2] = __fmaf_rn(ps[r], l.z, y[r][4 * c4 + 2]);
                            y[r][4 * c4 + 3] = __fmaf_rn(ps[r], l.w, y[r][4 * c4 + 3]);
                        }
                    }
                }
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const double fw = f * (double)wi[r];
#pragma unroll
                    for (int c = 0; c < 32; ++c)
                        if (mi[r] >> c & 1u) q[c] += fw * (double)y[r][c];
                }
            }
        }
        if (diag) {  // remove the i == j terms: a_ic w_i^2 psi_ii, halved like the rest of the diagonal tile
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const double s = 0.5 * (double)wi[r] * (double)grid_term(1.0f, wi[r], magic);
#pragma unroll
                for (int c = 0; c < 32; ++c)
                    if (mi[r] >> c & 1u) q[c] -= s;
            }
        }
    }
    // block reduction, fixed order
    __shared__ double s_q[kThreads / 32][32];
    __syncthreads();
#pragma unroll
    for (int c = 0; c < 32; ++c) {
        const double t = warp_sum(q[c]);
        if ((tid & 31) == 0) s_q[tid >> 5][c] = t;
    }
    __syncthreads();
    if (tid < 32) {
        double s = 0.0;
#pragma unroll
        for (int w = 0; w < kThreads / 32; ++w) s += s_q[w][tid];
        partialQ[(long long)blockIdx.x * 32 + tid] = s;
    }
}

// out[c] = sum over blocks b (in order) of partials[b * ncol + c].
__global__ void k_reduce_cols(const double *__restrict__ partials, int nblk, int ncol, double *__restrict__ out)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= ncol) return;
    double s = 0.0;
    for (int b = 0; b < nblk; ++b) s += partials[(long long)b * ncol + c];
    out[c] = s;
}

// R_c = sum_i a_ic w_i r_i and W_c = sum_i a_ic w_i for the 32 columns of mask word g = blockIdx.y, r_i the total
// row sum; slot 32 of each partial holds the all-rows sums (2S and the total weight).  Lane = column.
constexpr int kRWCols = 33;
template <int C>
__global__ void __launch_bounds__(kThreads) k_perm_RW(const float *__restrict__ rec, int F, int dim,
                                                     const uint32_t *__restrict__ maskg, const double *__restrict__ rowsum,
                                                     long long npad, int nchunk, double *__restrict__ partials)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, g = blockIdx.y;
    const long long rows_per_chunk = (npad + nchunk - 1) / nchunk;
    const long long r0 = blockIdx.x * rows_per_chunk, r1 = min(npad, r0 + rows_per_chunk);
    double R = 0.0, W = 0.0, Rall = 0.0, Wall = 0.0;
    for (long long i = r0 + warp; i < r1; i += kThreads / 32) {
        const double w = (double)rec[i * F + dim];
        double r = 0.0;
#pragma unroll
        for (int c = 0; c < C; ++c) r += rowsum[(long long)c * npad + i];
        const uint32_t m = maskg[(long long)g * npad + i];
        const double wr = w * r;
        if (m >> lane & 1u) { R += wr; W += w; }
        Rall += wr;
        Wall += w;
    }
    __shared__ double s[kThreads / 32][2][kRWCols];
    s[warp][0][lane] = R;
    s[warp][1][lane] = W;
    if (lane == 0) { s[warp][0][32] = Rall; s[warp][1][32] = Wall; }
    __syncthreads();
    if (threadIdx.x < 2 * kRWCols) {
        const int which = threadIdx.x / kRWCols, col = threadIdx.x % kRWCols;
        double t = 0.0;
#pragma unroll
        for (int w = 0; w < kThreads / 32; ++w) t += s[w][which][col];
        // partials[g][chunk][which][col]
        partials[(((long long)g * nchunk + blockIdx.x) * 2 + which) * kRWCols + col] = t;
    }
}

// Class-pair sums from row sums: out[tile][c2] = sum_{i in tile} w_i rowsum[c2][i]  (tile = kPad rows, one class).
template <int C>
__global__ void __launch_bounds__(kThreads) k_class_sums(const float *__restrict__ rec, int F, int dim,
                                                        const double *__restrict__ rowsum, long long npad,
                                                        double *__restrict__ out)
{
    __shared__ double s[kThreads / 32][C];
    const long long base = (long long)blockIdx.x * kPad;
    double a[C];
#pragma unroll
    for (int c = 0; c < C; ++c) a[c] = 0.0;
    for (int k = threadIdx.x; k < kPad; k += kThreads) {
        const double w = (double)rec[(base + k) * F + dim];
#pragma unroll
        for (int c = 0; c < C; ++c) a[c] += w * rowsum[(long long)c * npad + base + k];
    }
#pragma unroll
    for (int c = 0; c < C; ++c) {
        const double t = warp_sum(a[c]);
        if ((threadIdx.x & 31) == 0) s[threadIdx.x >> 5][c] = t;
    }
    __syncthreads();
    if (threadIdx.x < C) {
        double t = 0.0;
#pragma unroll
        for (int w = 0; w < kThreads / 32; ++w) t += s[w][threadIdx.x];
        out[(long long)blockIdx.x * C + threadIdx.x] = t;
    }
}

// ------------------------------------------------------------------------------------------------ labels
// Radix select of the n-th smallest composite key per permutation, 8 bits per pass from the top (reading R4).
// state[p] = {prefix (the digits fixed so far), rank (0-based rank still to locate inside the prefix bucket)}.
struct SelState {
    unsigned long long prefix;
    long long rank;
};

__global__ void k_sel_init(SelState *st, int nperm, long long n_x)
{
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p < nperm) { st[p].prefix = 0ull; st[p].rank = n_x - 1; }
}

// pass d (0..7): histogram of digit d of the keys whose higher digits equal the prefix.
// grid = (event chunks, Philox groups): group blockIdx.y covers the global permutations 4 * (p0 / 4 + blockIdx.y) + q,
// q < 4, of which those inside [p0, p0 + nperm) are local permutation p - p0.
__global__ void __launch_bounds__(kThreads) k_sel_hist(long long N, int nperm, long long p0, uint32_t seed_lo, uint32_t seed_hi,
                                                      int pass, const SelState *__restrict__ st, unsigned int *__restrict__ hist,
                                                      int ev_per_thread)
{
    __shared__ unsigned int h[4][256];
    for (int k = threadIdx.x; k < 1024; k += kThreads) (&h[0][0])[k] = 0u;
    const long long p4 = (p0 >> 2) + blockIdx.y;
    unsigned long long pre[4];
    long long pl[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        pl[q] = 4 * p4 + q - p0;
        if (pl[q] < 0 || pl[q] >= nperm) pl[q] = -1;
        pre[q] = pl[q] >= 0 ? st[pl[q]].prefix : 0ull;
    }
    __syncthreads();
    const int shift = 56 - 8 * pass;
    const long long base = (long long)blockIdx.x * kThreads * ev_per_thread;
    for (int e = 0; e < ev_per_thread; ++e) {
        const long long i = base + (long long)e * kThreads + threadIdx.x;
        if (i >= N) break;
        uint64_t K[4];
        label_keys4((uint32_t)i, (uint32_t)p4, seed_lo, seed_hi, K);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            if (pl[q] < 0) continue;
            const bool match = pass == 0 || (K[q] >> (shift + 8)) == pre[q];
            if (match) atomicAdd(&h[q][(K[q] >> shift) & 255u], 1u);
        }
    }
    __syncthreads();
    for (int k = threadIdx.x; k < 1024; k += kThreads) {
        const int q = k >> 8;
        const unsigned int v = (&h[0][0])[k];
        if (v && pl[q] >= 0) atomicAdd(&hist[pl[q] * 256 + (k & 255)], v);
    }
}

// one warp per permutation: locate the bucket holding the wanted rank, extend the prefix, clear the histogram
__global__ void k_sel_pick(SelState *st, unsigned int *hist, int nperm)
{
    const int p = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (p >= nperm) return;
    unsigned int *h = hist + (long long)p * 256;
    long long c[8], tot = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k) { c[k] = h[lane * 8 + k]; tot += c[k]; }
    long long incl = tot;  // inclusive scan over lanes
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const long long t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
    }
    const long long excl = incl - tot, rank = st[p].rank;
    __syncwarp();
    if (rank >= excl && rank < incl) {  // exactly one lane
        long long cum = excl;
        int b = 7;
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            if (b == 7 && k < 7 && rank < cum + c[k]) b = k;
            if (b == 7 && k < 7) cum += c[k];
        }
        st[p].prefix = (st[p].prefix << 8) | (unsigned long long)(lane * 8 + b);
        st[p].rank = rank - cum;
    }
    __syncwarp();
#pragma unroll
    for (int k = 0; k < 8; ++k) h[lane * 8 + k] = 0u;
}

// After the four passes over the key32 half of the composites the wanted one lies in the bucket of the events whose key32
// equals the prefix: one event plus N / 2^32 expected others.  Instead of four more sweeps over the index half (each
// a Philox evaluation per event and four permutations), ONE sweep lists the bucket's events and k_sel_finish takes the
// rank-th smallest index among them -- the same K*_p.  cand[p][kSelCand]; a bucket that does not fit (cnt > kSelCand:
// not reachable for N < 2^31, expected bucket size <= 1.5) sets *overflow and the host falls back to the four sweeps.
constexpr int kSelCand = 64;
__global__ void __launch_bounds__(kThreads) k_sel_collect(long long N, int nperm, long long p0, uint32_t seed_lo, uint32_t seed_hi,
                                                         const SelState *__restrict__ st, unsigned int *__restrict__ cand_cnt,
                                                         uint32_t *__restrict__ cand, int ev_per_thread)
{
    const long long p4 = (p0 >> 2) + blockIdx.y;
    unsigned long long pre[4];
    long long pl[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        pl[q] = 4 * p4 + q - p0;
        if (pl[q] < 0 || pl[q] >= nperm) pl[q] = -1;
        pre[q] = pl[q] >= 0 ? st[pl[q]].prefix : 0ull;
    }
    const long long base = (long long)blockIdx.x * kThreads * ev_per_thread;
    for (int e = 0; e < ev_per_thread; ++e) {
        const long long i = base + (long long)e * kThreads + threadIdx.x;
        if (i >= N) break;
        uint64_t K[4];
        label_keys4((uint32_t)i, (uint32_t)p4, seed_lo, seed_hi, K);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            if (pl[q] < 0 || (K[q] >> 32) != pre[q]) continue;
            const unsigned int slot = atomicAdd(&cand_cnt[pl[q]], 1u);
            if (slot < (unsigned)kSelCand) cand[pl[q] * kSelCand + slot] = (uint32_t)i;
        }
    }
}
// one thread per permutation; *overflow != 0 afterwards: some bucket did not fit and NO state may be used
__global__ void k_sel_finish(SelState *st, unsigned int *__restrict__ cand_cnt, const uint32_t *__restrict__ cand, int nperm, int *overflow)
{
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= nperm) return;
    const unsigned int cnt = cand_cnt[p];
    cand_cnt[p] = 0u;  // clean for the next call
    if (cnt > (unsigned)kSelCand) { atomicOr(overflow, 1); return; }
    const uint32_t *c = cand + (long long)p * kSelCand;
    const long long rank = st[p].rank;
    for (unsigned int a = 0; a < cnt; ++a) {
        long long below = 0;
        for (unsigned int b = 0; b < cnt; ++b) below += c[b] < c[a] ? 1 : 0;   // indices are distinct
        if (below == rank) {
            st[p].prefix = (st[p].prefix << 32) | (unsigned long long)c[a];
            st[p].rank = 0;
            return;
        }
    }
    atomicOr(overflow, 2);  // rank outside the bucket: cannot happen (the histogram passes counted these events)
}

// Writes label words.  After the eight passes st[p].prefix is the n-th smallest composite K*_p; a_ip = (K_ip <= K*_p).
// Column c of the output: c < col_off is the observed labelling (i < n_x), else permutation c - col_off.
// Output word for pooled event i and word index g: out[g * stride_g + pos(i) * stride_i].
struct LabelOut {
    long long stride_g, stride_i;
    int nseg;                          // pooled index -> row position, by segments
    long long seg_first[kMaxCls + 1];  // first pooled index of each segment
    long long seg_pos[kMaxCls];        // row position of that first index
};
__global__ void __launch_bounds__(kThreads) k_label_write(long long N, long long n_x, int nperm, long long p0, int col_off,
                                                         int nwords, uint32_t seed_lo, uint32_t seed_hi,
                                                         const SelState *__restrict__ st, LabelOut L,
                                                         uint32_t *__restrict__ out)
{
    const long long i = blockIdx.x * (long long)kThreads + threadIdx.x;
    const int g = blockIdx.y;
    if (i >= N) return;
    uint32_t word = 0u;
    uint64_t K[4];
    long long have_p4 = -1;
    for (int b = 0; b < 32; ++b) {
        const int c = 32 * g + b;
        if (c < col_off) { if (i < n_x) word |= 1u << b; continue; }
        const int p = c - col_off;
        if (p >= nperm) break;
        const long long pg = p0 + p;  // global permutation index
        if ((pg >> 2) != have_p4) { have_p4 = pg >> 2; label_keys4((uint32_t)i, (uint32_t)have_p4, seed_lo, seed_hi, K); }
        if (K[pg & 3] <= st[p].prefix) word |= 1u << b;
    }
    long long pos = i;
    for (int s = 0; s < L.nseg; ++s)
        if (i >= L.seg_first[s] && i < L.seg_first[s + 1]) pos = L.seg_pos[s] + (i - L.seg_first[s]);
    (void)nwords;
    out[(long long)g * L.stride_g + pos * L.stride_i] = word;
}

// ------------------------------------------------------------------------------------------------ Sect. 5 split
// positive[i] = 1 iff C = pB . (pC x pD) > 0 (or -C > 0 when conj), fp64 with the oracle's operation order and no
// contraction, so the sign agrees bit for bit (reading R11: C == 0 is negative).
__device__ __forceinline__ int triple_positive(const double *b, const double *c, const double *d, int conj)
{
    const double cx = __dsub_rn(__dmul_rn(c[1], d[2]), __dmul_rn(c[2], d[1]));
    const double cy = __dsub_rn(__dmul_rn(c[2], d[0]), __dmul_rn(c[0], d[2]));
    const double cz = __dsub_rn(__dmul_rn(c[0], d[1]), __dmul_rn(c[1], d[0]));
    const double C = __dadd_rn(__dadd_rn(__dmul_rn(b[0], cx), __dmul_rn(b[1], cy)), __dmul_rn(b[2], cz));
    const double v = conj ? -C : C;
    return v > 0.0 ? 1 : 0;
}

// separate pB, pC, pD arrays [n][3] (stride 3) or one [n][3][3] array (stride 9, offsets 0, 3, 6)
__global__ void k_podd_flags(const double *pB, const double *pC, const double *pD, long long n, int stride, int conj,
                             uint8_t *positive, unsigned long long *count)
{
    const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    int f = 0;
    if (i < n) {
        f = triple_positive(pB + i * stride, pC + i * stride, pD + i * stride, conj);
        positive[i] = (uint8_t)f;
    }
    const unsigned int b = __ballot_sync(0xffffffffu, f);
    if ((threadIdx.x & 31) == 0 && b) atomicAdd(count, (unsigned long long)__popc(b));
}

// Stable partition of the pooled source events into the four class segments of the P-odd layout:
// layout class 0 = I (D, C_T > 0), 1 = IV (Dbar, -Cbar_T <= 0), 2 = II, 3 = III; A = {0, 1}, B = {2, 3}.
__global__ void k_podd_classes(long long N, long long n, const uint8_t *__restrict__ posx, const uint8_t *__restrict__ posb,
                               uint8_t *__restrict__ cls)
{
    const long long s = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (s >= N) return;
    cls[s] = s < n ? (posx[s] ? 0 : 2) : (posb[s - n] ? 3 : 1);
}
// Stable four-way partition of the indices 0 .. N-1 by cls[s] (k_part_count, k_part_scan, k_part_scatter).
constexpr int kPartBlock = 1024;
__global__ void __launch_bounds__(kPartBlock) k_part_count(long long N, const uint8_t *__restrict__ cls, int *__restrict__ blk_cnt)
{
    __shared__ int cnt[4];
    if (threadIdx.x < 4) cnt[threadIdx.x] = 0;
    __syncthreads();
    const long long s = blockIdx.x * (long long)kPartBlock + threadIdx.x;
    if (s < N) atomicAdd(&cnt[cls[s]], 1);
    __syncthreads();
    if (threadIdx.x < 4) blk_cnt[blockIdx.x * 4 + threadIdx.x] = cnt[threadIdx.x];
}
// single thread block: exclusive scan over blocks per class; totals[4]
__global__ void k_part_scan(int nblk, int *__restrict__ blk_cnt, long long *__restrict__ totals)
{
    if (threadIdx.x < 4) {
        long long run = 0;
        for (int b = 0; b < nblk; ++b) {
            const int v = blk_cnt[b * 4 + threadIdx.x];
            blk_cnt[b * 4 + threadIdx.x] = (int)run;
            run += v;
        }
        totals[threadIdx.x] = run;
    }
}
// src[seg_pos[c] + rank] = s, ranks in increasing s (stable)
__global__ void __launch_bounds__(kPartBlock) k_part_scatter(long long N, const uint8_t *__restrict__ cls,
                                                            const int *__restrict__ blk_off, const long long *__restrict__ seg_pos,
                                                            int *__restrict__ src)
{
    __shared__ int warp_cnt[kPartBlock / 32][4];
    const long long s = blockIdx.x * (long long)kPartBlock + threadIdx.x;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int c = s < N ? (int)cls[s] : -1;
    unsigned int bal[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) bal[k] = __ballot_sync(0xffffffffu, c == k);
    if (lane < 4) warp_cnt[warp][lane] = __popc(bal[lane]);
    __syncthreads();
    if (c >= 0) {
        int rank = __popc(bal[c] & ((1u << lane) - 1u));
        for (int w = 0; w < warp; ++w) rank += warp_cnt[w][c];
        src[seg_pos[c] + blk_off[blockIdx.x * 4 + c] + rank] = (int)s;
    }
}
__global__ void k_fill_int(int *p, long long n, int v)
{
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) p[i] = v;
}

// ---- Eq. 3 permutation test (one all-pairs pass per permutation over re-ordered records) ---------------------
// Sources: the pooled source index s of et_T_bkg's staging, x side = [x (n) ; bx (bs)], xbar side = [xbar (nbar) ;
// bxbar (bsbar)].  Main pool index: x[k] -> k, xbar[k] -> n + k; background pool index: bx[k] -> k, bxbar[k] -> bs + k.
struct BkgPermParams {
    long long n, nbar, bs, bsbar;
    long long pos0[4];   // first record row of the identity layout's class segments (X, Bx, Xbar, Bxbar)
    uint32_t seedm_lo, seedm_hi, seedb_lo, seedb_hi;
};
// cls[s] = class (X', Bx', Xbar', Bxbar') = (0, 1, 2, 3) that permutation pg (global index; `sm`, `sb` its select states
// for the main and the background pool) gives source event s, s running over X | Bx | Xbar | Bxbar in input order (the
// class segments of the identity layout).  The stable four-way partition k_part_* then lists, class by class and in
// source order, which source event every row of the permuted layout holds; the class sizes are those of the identity
// layout (the labels preserve sample sizes), so the layout never changes.
__global__ void __launch_bounds__(kThreads) k_bkg_class(BkgPermParams P, long long pg, const SelState *__restrict__ sm,
                                                       const SelState *__restrict__ sb, uint8_t *__restrict__ cls)
{
    const long long Nx = P.n + P.bs, Ntot = Nx + P.nbar + P.bsbar;
    const long long s = blockIdx.x * (long long)kThreads + threadIdx.x;
    if (s >= Ntot) return;
    bool bkg;
    long long idx;  // index in its pool
    if (s < Nx) { bkg = s >= P.n; idx = bkg ? s - P.n : s; }
    else {
        const long long t = s - Nx;
        bkg = t >= P.nbar;
        idx = bkg ? P.bs + (t - P.nbar) : P.n + t;
    }
    uint64_t K[4];
    label_keys4((uint32_t)idx, (uint32_t)(pg >> 2), bkg ? P.seedb_lo : P.seedm_lo, bkg ? P.seedb_hi : P.seedm_hi, K);
    const bool in_x = K[pg & 3] <= (bkg ? sb->prefix : sm->prefix);
    cls[s] = (uint8_t)((in_x ? 0 : 2) + (bkg ? 1 : 0));
}
// ---- guard-band escalation (exact p-value) ------------------------------------------------
// Class of pooled (label) index i for the re-evaluation of permutation p: 2 (1 - a_obs) + (1 - a_perm), i.e.
// 0 = in X of both labellings, 1 = X observed / Xbar permuted, 2 = Xbar observed / X permuted, 3 = Xbar of both.
// a_perm by the rule of reading R4 from the select state of p (K_ip <= K*_p).
__global__ void __launch_bounds__(kThreads) k_esc_class(long long N, long long n_x, long long pg, uint32_t seed_lo, uint32_t seed_hi,
                                                       const SelState *__restrict__ st, uint8_t *__restrict__ cls)
{
    const long long i = blockIdx.x * (long long)kThreads + threadIdx.x;
    if (i >= N) return;
    uint64_t K[4];
    label_keys4((uint32_t)i, (uint32_t)(pg >> 2), seed_lo, seed_hi, K);
    const int a_perm = K[pg & 3] <= st->prefix, a_obs = i < n_x;
    cls[i] = (uint8_t)(2 * (1 - a_obs) + (1 - a_perm));
}
// rec2[row] = rec[pos(src[row])]: src[row] is the pooled (label) index that the escalation layout puts into `row`
// (-1: padding, zero record), pos() its row in the records of the call's own layout (class segments of L).
__global__ void k_esc_gather(const float4 *__restrict__ rec, const int *__restrict__ src, long long npad2, int F4, LabelOut L,
                             float4 *__restrict__ rec2)
{
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < npad2 * F4; k += (long long)gridDim.x * blockDim.x) {
        const long long row = k / F4;
        const int q = (int)(k % F4);
        const long long i = src[row];
        float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
        if (i >= 0) {
            long long pos = i;
            for (int s = 0; s < L.nseg; ++s)
                if (i >= L.seg_first[s] && i < L.seg_first[s + 1]) pos = L.seg_pos[s] + (i - L.seg_first[s]);
            v = rec[pos * F4 + q];
        }
        rec2[k] = v;
    }
}

// count = #{T_p > T_obs}, near = #{|T_p - T_obs| <= guard or T_p not finite}; one block
__global__ void __launch_bounds__(256) k_count_gt(const double *__restrict__ T, int nperm, double Tobs, double guard, long long *__restrict__ out)
{
    __shared__ unsigned long long s_cnt, s_near;
    if (threadIdx.x == 0) { s_cnt = 0ull; s_near = 0ull; }
    __syncthreads();
    unsigned long long c = 0, nr = 0;
    for (int p = threadIdx.x; p < nperm; p += blockDim.x) {
        const double t = T[p];
        if (!isfinite(t)) { nr += 1; continue; }
        if (t > Tobs) c += 1;
        if (fabs(t - Tobs) <= guard) nr += 1;
    }
    atomicAdd(&s_cnt, c);
    atomicAdd(&s_near, nr);
    __syncthreads();
    if (threadIdx.x == 0) { out[0] = (long long)s_cnt; out[1] = (long long)s_near; }
}

// gather of the listed rows of rowsum (test hook et_row_sums)
__global__ void k_gather_rows(const double *__restrict__ rowsum, long long npad, const long long *__restrict__ pos, long long nrows,
                              int C, double *__restrict__ out)
{
    const long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (k >= nrows) return;
    for (int c = 0; c < C; ++c) out[c * nrows + k] = rowsum[(long long)c * npad + pos[k]];
}

}  // namespace et
