// et_device.cuh -- device-side building blocks shared by the kernels of libet.so.
// Not shared with oracle/ (the oracle is a separate plain-C translation unit).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace et {

constexpr int kThreads = 256;   // threads per CTA in every all-pairs kernel
constexpr int kTileJ = 256;     // j rows staged in shared memory per step
constexpr int kPad = 1024;      // every class segment is padded to a multiple of this many rows
constexpr int kMaxCls = 4;      // classes in the pooled layout (2 for X/Xbar, 4 for the Sect. 5 split)
constexpr int kSumSlots = 16;   // class-pair block sums, slot c1 * 4 + c2 with c1 <= c2
// The CUDA-core PERMUTATION kernels (k_pairs_rows, k_perm32) keep an fp32 partial sum over this many pairs only, and the
// terms they add are first rounded to a fixed grid on which such a partial sum is exact (grid_term, et_kernels.cuh).  Why: an
// fp32 accumulator of size A drops the part of every addend below ulp(A) / 2; psi has most of its mass near 0 (far
// pairs, density ~ 1 / psi), so the loss is a bias proportional to ulp(A) -- and the accumulators of a random labelling
// (half the j of a block) are half as large as those of the row sums r_i and of the contiguous observed labelling.
// Measured against the oracle (tests/test_gpu_parity.py::test_error_model_of_the_decision): with 256 plain fp32 adds per
// partial every T_p sat +7e-9 above its oracle value at sigma = 0.3 while T_obs was exact (2e-8 of the term scale, far
// inside the 1e-6 tolerance of T but 30 sigma of the error model that certifies T_p > T_obs); 32 adds left +5e-10; on the
// grid Q_p, R_p and S are exact sums of the same numbers and the offset is gone, as on the tensor-core path.
// (k_pairs_T sums whole blocks of contiguous classes: every class pair carries the same relative loss, which cancels in
// T like the 6e-8 bias of ex2.approx.)
constexpr int kFlushJ = 32;

// Floats per event record in the pooled layout: dim coordinates, then the weight, zero padded to a float4 multiple.
__host__ __device__ constexpr int rec_floats(int dim) { return (dim + 1 + 3) / 4 * 4; }

// 2^x by one MUFU.EX2 (ex2.approx.ftz.f32).  psi = 2^(-|u_i - u_j|^2) with u the pre-scaled coordinates.
__device__ __forceinline__ float ex2_approx(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// psi_ij of PAPER.md:71 in the pre-scaled coordinates u = (x - c) * sqrt(log2(e) / (2 sigma^2)).
// The instruction sequence is spelled out with _rn intrinsics so that every kernel of the library rounds every
// pair identically (S, r_i and Q_p must be sums of the SAME psi values: DESIGN.md "consistency").
template <int D>
__device__ __forceinline__ float psi_pair(const float (&ui)[D], const float *__restrict__ uj)
{
    float d = __fsub_rn(ui[0], uj[0]);
    float e = __fmul_rn(d, d);
#pragma unroll
    for (int k = 1; k < D; ++k) {
        d = __fsub_rn(ui[k], uj[k]);
        e = __fmaf_rn(d, d, e);
    }
    return ex2_approx(-e);
}

// Row-major enumeration of the upper triangle (I <= J) of an nT x nT tile grid.
__device__ __forceinline__ void unit_to_pair(long long u, int nT, int &I, int &J)
{
    const double b = 2.0 * nT + 1.0;
    int i = (int)((b - sqrt(b * b - 8.0 * (double)u)) * 0.5);
    if (i < 0) i = 0;
    if (i > nT - 1) i = nT - 1;
    auto off = [nT](long long r) { return r * nT - r * (r - 1) / 2; };
    while (i + 1 < nT && off(i + 1) <= u) ++i;
    while (i > 0 && off(i) > u) --i;
    I = i;
    J = i + (int)(u - off(i));
}

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Philox4x32-10 (Salmon et al., SC'11), the label generator fixed by reading R4.
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              uint32_t k0, uint32_t k1, uint32_t (&out)[4])
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// Composite sort key of pooled event i in permutation p (reading R4): (key32 << 32) | i.
__device__ __forceinline__ void label_keys4(uint32_t i, uint32_t p4, uint32_t seed_lo, uint32_t seed_hi, uint64_t (&K)[4])
{
    uint32_t o[4];
    philox4x32_10(i, 0u, p4, 0u, seed_lo, seed_hi, o);
#pragma unroll
    for (int q = 0; q < 4; ++q) K[q] = ((uint64_t)o[q] << 32) | i;
}

}  // namespace et
