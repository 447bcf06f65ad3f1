// et_tc.cuh -- K-PERM-TC: the permutation sums of SURVEY 8(a) H5 on the sm_100a tensor cores (tcgen05, kind::i8).
//
// Identity: with label columns a_jc in {0,1} and
//   Y_ic = sum_{j > i} Psi_ij a_jc,            Psi_ij = w_j psi_ij   (w = 1 when unweighted),
// the three sums every column needs are row reductions of Y:
//   Q_c = sum_{i<j} w_i w_j psi_ij a_ic a_jc           = sum_i a_ic w_i Y_ic
//   R_c = sum_{i<j} w_i w_j psi_ij (a_ic + a_jc)       = sum_i real_i w_i Y_ic + sum_i a_ic w_i Y_i,ones
//   S   = sum_{i<j} w_i w_j psi_ij                     = Q of the all-ones column
// and S_xx = Q, S_bb = S - R + Q, S_xb = R - 2Q.  Y = Psi A is a GEMM whose left operand is
// never stored.  A cluster of two CTAs (one SM pair) works on a 256-row tile; per K block of KB j (Geo below: 128 or 96)
// each CTA evaluates its 128 x KB tile of psi in fp32 (packed FFMA2 + MUFU.EX2, KB / 8 producer warps, 4 rows x 8 j per
// thread; the j side comes as pre-formatted pair records that a loader warp bulk-copies into a shared-memory ring),
// quantises Psi_ij = w_j psi_ij to a 15-bit fixed-point integer v = lo + 128 hi (lo = v & 255, hi = 2 (v >> 8); see
// kMagicUnsigned below), writes the two digit tiles into its shared memory as K chunks of 32 bytes in the UMMA K-major
// SWIZZLE_32B layout, and expands ITS HALF of the label columns from the bit masks into the B tile (bytes a and 128 a,
// MN-major SWIZZLE_128B).  One thread of the leader CTA issues tcgen05.mma.cta_group::2.kind::i8 (M = 256, N = 256,
// K = 32): the pair's tensor cores read A from their own SM and each half of B from one SM of the pair, so a label byte
// is written and read once per 256 rows instead of once per 128.  At config 4 the tensor pipe is 74 % busy, the producers
// are latency-bound and the board sits at its power cap (profiles/r02_README.md).  Accumulation is
// ONE int32 per column in TMEM (all 512 columns of each SM).  Integer accumulation is exact, so S, R and Q are sums of the
// SAME quantised Psi whatever the schedule (hard part 3 "consistency"), and the unweighted result is
// bit-reproducible.
//
// Columns of one launch (512): 0 = observed labelling, 1 = second labelling (P-even grouping of Sect. 5, else a copy
// of column 0), 2 = all ones, 3.. = 509 permutations.  Inside a 32-column mask word the B tile / TMEM column p holds
// label bit beta(p) = (p >> 2) + 8 (p & 3), so that four label bytes come out of one shift and one mask.
#pragma once
#include <type_traits>

#include "et_kernels.cuh"

namespace et {
namespace tc {

constexpr int kTM = 128;                 // rows (i) per CTA = UMMA M / 2
constexpr int kTM2 = 2 * kTM;            // rows per cluster (work unit)
constexpr int kCols = 512;               // label columns per launch (2 accumulators of N = 256)
constexpr int kSpecial = 3;              // observed, second labelling, ones
constexpr int kPermsPerChunk = kCols - kSpecial;
constexpr int kWordsPerChunk = kCols / 32;
constexpr int kMaxRecSlots = 4;
constexpr int kMaxDimTC = 8;          // = ET_MAX_DIM (include/et.h)
// float4 per pair record: dim + 1 float2 entries, padded to an even count
__host__ __device__ constexpr int pair_rec_f4(int dim) { return (dim + 2) / 2; }

// Geometry of the kernel: K blocks of KB j (KB / 32 UMMA K steps), PW producer warps (a thread evaluates 4 rows x 8 j of
// the 128 x KB psi tile of its CTA: PW = KB / 8), ST shared-memory stages.  Two are built:
//   Geo<96, 12, 3>:  16 warps (12 producers, MMA, loader, two label helpers) x 128 registers, three 72 KB stages.
//   Geo<128, 16, 2>: 20 warps x 96 registers, two 96 KB stages: a fourth producer warp per scheduler hides more of the
//                    producers' latency (profiles/r02_README.md: -4.6 % at config 4, same at dim = 2), but the i rows of
//                    dim >= 6 no longer fit the registers (dim = 8: +75 %).  run_perm_tc takes it for dim <= 5.
template <int KB, int PW, int ST>
struct Geo {
    static constexpr int kKB = KB;                  // j per K block
    static constexpr int kProducerWarps = PW;
    static constexpr int kStages = ST;
    static constexpr int kRowsPerThread = kTM * KB / 8 / (PW * 32);  // 4
    static constexpr int kEpiWarps = PW / 4;                         // warps per TMEM lane quarter
    static constexpr int kEpiGroups = (16 + kEpiWarps - 1) / kEpiWarps;  // most 32-column groups a warp reads in the epilogue
    __host__ __device__ static constexpr int epi_first(int e) { return 16 * e / kEpiWarps; }  // groups [epi_first(e), epi_first(e + 1)) of warp row e
    static constexpr int kProducers = PW * 32;
    static constexpr int kHelperWarps = 2;              // label helpers: the B tile of the second accumulator (k_perm_tc)
    static constexpr int kThreadsTC = kProducers + 64 + 32 * kHelperWarps;  // + the MMA warp + the record loader warp + the helpers
    static_assert(KB % (16 * kHelperWarps) == 0, "whole 8-j groups per helper warp");
    static constexpr int kABytes = 2 * kTM * KB;        // hi and lo digit tiles
    static constexpr int kBPlane = KB * 128;            // one plane of this CTA's half of B: KB j x 128 columns
    static constexpr int kBBytes = 2 * 2 * kBPlane;     // [q 2][digit 2][plane]
    static constexpr int kStageBytes = kABytes + kBBytes;
    // ring of j pair-record blocks (KB / 2 pairs each), filled by bulk copies (see the loader)
    __host__ __device__ static constexpr int rec_slots(int dim) { return pair_rec_f4(dim) <= 3 ? 4 : 2; }
    __host__ __device__ static constexpr int rec_slot_bytes(int dim) { return (KB / 2) * pair_rec_f4(dim) * 16; }
    __host__ __device__ static constexpr int smem_tc(int dim) { return ST * kStageBytes + rec_slots(dim) * rec_slot_bytes(dim) + 1024 /*alignment slack*/; }
    // K blocks per unit: |Y| <= 32767 * KB * kMaxUnitKB < 2^31 (660 for KB = 96: 2 076 117 120; 511 for KB = 128).  Longer
    // units mean fewer epilogues and pipeline drains (512 -> 1000 blocks of 64 j measured -1.2 % at config 2 and -0.9 % at
    // config 4, identical integer sums).
    static constexpr int kMaxUnitKB = 2147483647ll / (32767ll * KB) > 660 ? 660 : (int)(2147483647ll / (32767ll * KB));
    static_assert(32767ll * KB * kMaxUnitKB < 2147483648ll, "int32 accumulator headroom");
    static_assert(PW * 8 == KB && PW % 4 == 0, "one producer warp per 8 j, whole warp rows in the epilogue");
};
using Geo96 = Geo<96, 12, 3>;
using Geo128 = Geo<128, 16, 2>;
// Quantisation of Psi_ij = w_j psi_ij to the 15-bit grid of step 1 / sc: f = fma.rz(psi, 256 sc w_j, M + 128) with
// M = 2^23 holds, in mantissa bits 8..22, v = floor(sc Psi + 1/2), 0 <= v <= 32767 (weights >= 0).  With signed weights
// M = 1.5 * 2^23 and the same bits hold 16384 + v, |v| <= 16383.  The two operand digits are BYTES 1 and 2 of f:
// lo = v & 255 (u8, label plane a) and hi = 2 (v >> 8) (u8 <= 254; signed: 2 byte2 - 128 as s8; label plane 128 a),
// 128 hi + lo = v.
//
// Plain round-to-nearest, NO dither -- measured on the B200 (12 samples each, n = nbar = 2e4 .. 3.2e5, sigma 0.1 .. 0.5,
// errors in units of the independent-error model sigma of T):
//   * round to nearest:                      T_obs 0.2-0.6, T_p 0.4-0.7 at every size.  The rounding error is the same
//     function of psi for every pair, i.e. a tiny perturbation of the distance function, consistent between T_obs and
//     every T_p.  Cost: the psi values below half a step are lost, -0.005 steps per pair on the Dalitz samples, so each
//     BLOCK SUM is low by 7e-7 (unit weights) to 2.6e-6 (signed weights) of itself -- the same fraction of S_xx, S_bb
//     and S_xb, which cancels in T (1/2 + 1/2 - 1 = 0).
//   * dither levels that are a constant of the thread (2 levels: the earlier round-to-16-bits + alternating halving;
//     or 32 levels over the lanes): unbiased block sums, T_p fine (0.9-1.0), but T_obs 2-10 and GROWING like sqrt N.
//     Below one step v is 0 or 1 by comparing sc Psi with the level; a row that meets only its thread's few levels keeps
//     a bias of its own, random over the rows; random labellings average it (row weights ~ sqrt N), the contiguous
//     OBSERVED labelling sums it coherently (row weights ~ N).  Rotating the levels from K block to K block only
//     halves it.  A per-pair pseudo-random level would cost one more instruction per psi and double the variance.
// The decision T_p > T_obs is what the path is for, so the rounding is the plain one; kQuantVar is its error variance
// in steps^2 (uniform error), used by the guard band.
constexpr float kMagicUnsigned = 8388608.0f, kMagicSigned = 12582912.0f;
constexpr double kQuantVar = 1.0 / 12.0;
constexpr double kScaleUnsigned = 32766.0, kScaleSigned = 16382.0;  // floor(sc Psi + 1/2) <= 32767 with the fp32 slack of sc w_j

// label bit held by byte / TMEM column p of a 32-column word
__host__ __device__ constexpr int beta(int p) { return (p >> 2) + 8 * (p & 3); }

struct Unit {
    int I;         // 256-row tile
    int kb_begin;  // first K block (Geo::kKB j each), >= the block that holds the tile's first row
    int kb_end;
    int pad;
};

// ---- PTX wrappers ------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ uint64_t pack2(float a, float b)
{
    uint64_t r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b));
    return r;
}
__device__ __forceinline__ void unpack2(uint64_t v, float &a, float &b) { asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); }
__device__ __forceinline__ uint64_t add2(uint64_t a, uint64_t b)
{
    uint64_t r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ uint64_t mul2(uint64_t a, uint64_t b)
{
    uint64_t r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ uint64_t fma2(uint64_t a, uint64_t b, uint64_t c)
{
    uint64_t r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}
// round-toward-zero FMA: with the magic constant the sum is positive, so the low mantissa bits hold floor(a b) + 2
__device__ __forceinline__ uint64_t fma2_rz(uint64_t a, uint64_t b, uint64_t c)
{
    uint64_t r;
    asm("fma.rz.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    uint32_t done = 0;
    while (!done) {
        asm volatile(
            "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}\n"
            : "=r"(done)
            : "r"(smem_u32(bar)), "r"(parity)
            : "memory");
    }
}
__device__ __forceinline__ void mbar_wait_a(uint32_t bar_addr, uint32_t parity)
{
    uint32_t done = 0;
    while (!done) {
        asm volatile(
            "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}\n"
            : "=r"(done)
            : "r"(bar_addr), "r"(parity)
            : "memory");
    }
}
__device__ __forceinline__ void umma_commit(uint64_t *bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// ---- cluster (CTA pair) forms ------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t cluster_ctarank()
{
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_sync_all()
{
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// shared::cluster address of `local` (a shared::cta address) in the CTA of rank `rank`
__device__ __forceinline__ uint32_t mapa_rank(uint32_t local, uint32_t rank)
{
    uint32_t r;
    asm("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(local), "r"(rank));
    return r;
}
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t cluster_addr)
{
    // default semantics (release at CTA scope), as the CUTLASS cluster barriers use: the data the peer's MMAs read was
    // published to the async proxy by this thread's fence.proxy.async; a .release.cluster here costs a MEMBAR.GPU +
    // L1 invalidate per arrive (profiles/r01b)
    asm volatile("mbarrier.arrive.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}
__device__ __forceinline__ void mbar_wait_cluster(uint64_t *bar, uint32_t parity)
{
    uint32_t done = 0;
    while (!done) {
        asm volatile(
            "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}\n"
            : "=r"(done)
            : "r"(smem_u32(bar)), "r"(parity)
            : "memory");
    }
}
// arrives (count 1) on the barrier at this shared-memory offset in BOTH CTAs of the pair once all prior MMAs are done
__device__ __forceinline__ void umma_commit_pair(uint64_t *bar)
{
    asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(smem_u32(bar)),
                 "h"((uint16_t)3)
                 : "memory");
}
__device__ __forceinline__ void umma_i8_pair(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::2.kind::i8 [%0], %1, %2, %3, p;\n\t}\n" ::"r"(tmem_d),
        "l"(da), "l"(db), "r"(idesc), "r"(accumulate)
        : "memory");
}
// bulk copy global -> this CTA's shared memory, completion counted in bytes on an mbarrier (one thread issues)
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint64_t *bar)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst), "l"(src), "r"(bytes),
                 "r"(smem_u32(bar))
                 : "memory");
}
// shared-memory accesses by 32-bit shared-space address (immediate offsets fold into the instruction)
__device__ __forceinline__ float4 lds128(uint32_t a)
{
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a));
    return v;
}
__device__ __forceinline__ void sts64(uint32_t a, uint2 v) { asm volatile("st.shared.v2.b32 [%0], {%1, %2};" ::"r"(a), "r"(v.x), "r"(v.y) : "memory"); }
__device__ __forceinline__ void sts128(uint32_t a, uint4 v)
{
    asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(a), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
// hides a loop-invariant value from the optimiser (see the producer loop)
__device__ __forceinline__ int keep(int x) { asm volatile("" : "+r"(x)); return x; }
__device__ __forceinline__ float keep(float x) { asm volatile("" : "+f"(x)); return x; }
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

// UMMA shared-memory descriptor (sm_100): start >> 4, LBO >> 4 at bit 16, SBO >> 4 at bit 32, version 1 at bit 46,
// layout type at bit 61 (2 = SWIZZLE_128B, 4 = SWIZZLE_64B).
__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes, uint32_t layout)
{
    uint64_t d = 0;
    d |= (uint64_t)((saddr >> 4) & 0x3fff);
    d |= (uint64_t)((lbo_bytes >> 4) & 0x3fff) << 16;
    d |= (uint64_t)((sbo_bytes >> 4) & 0x3fff) << 32;
    d |= (uint64_t)1 << 46;
    d |= (uint64_t)layout << 61;
    return d;
}
// kind::i8 instruction descriptor: D = s32, A u8/s8 K-major, B u8 MN-major, M = 256 (the CTA pair), N = 256.
__host__ __device__ constexpr uint32_t umma_idesc_i8(bool a_signed)
{
    return (2u << 4) | ((a_signed ? 1u : 0u) << 7) | (0u << 10) | (0u << 15) | (1u << 16) | ((256u >> 3) << 17) | ((256u >> 4) << 24);
}
__device__ __forceinline__ void umma_i8(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n\t}\n" ::"r"(tmem_d),
        "l"(da), "l"(db), "r"(idesc), "r"(accumulate)
        : "memory");
}
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&v)[32])
{
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, %17, %18, %19, "
        "%20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]), "=r"(v[9]),
          "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]), "=r"(v[17]), "=r"(v[18]),
          "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]),
          "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
        : "r"(taddr));
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ uint32_t tmem_ld1(uint32_t taddr)
{
    uint32_t v;
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x1.b32 {%0}, [%1];" : "=r"(v) : "r"(taddr));
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
    return v;
}

// Sum over the 32 lanes of x[b] for every b: lane L returns the total of element L (31 shuffles).
template <typename T>
__device__ __forceinline__ T lane_transpose_sum(T (&x)[32], int lane)
{
#pragma unroll
    for (int s = 16; s >= 1; s >>= 1) {
        const bool upper = (lane & s) != 0;
#pragma unroll
        for (int k = 0; k < s; ++k) {
            const T send = upper ? x[k] : x[k + s];
            const T keep = upper ? x[k + s] : x[k];
            x[k] = keep + __shfl_xor_sync(0xffffffffu, send, s);
        }
    }
    return x[0];
}

// Pair records of the j side: recP[pair][entry] float2, entry k < D = (-u_{2 pair, k}, -u_{2 pair + 1, k}), entry D =
// (s, s') with s = 256 sc w_j (the quantisation scale times the weight), zero padded to pair_rec_f4(D) float4.  With the
// i rows as scalar-broadcast operands (u_ik, u_ik) of the packed instructions, d = u_i + (-u_j) and Psi = 2^(-e) s + magic are packed FADD2 / FFMA2 over two j.
template <int D>
__global__ void __launch_bounds__(kThreads) k_pair_records(const float *__restrict__ rec, long long npairs, float sc, float4 *__restrict__ recP)
{
    constexpr int F = rec_floats(D), NLD = pair_rec_f4(D);
    const long long pr = blockIdx.x * (long long)kThreads + threadIdx.x;
    if (pr >= npairs) return;
    float a[F], b[F], o[4 * NLD];
#pragma unroll
    for (int q = 0; q < F / 4; ++q) {
        const float4 ta = reinterpret_cast<const float4 *>(rec + 2 * pr * F)[q], tb = reinterpret_cast<const float4 *>(rec + (2 * pr + 1) * F)[q];
        a[4 * q] = ta.x; a[4 * q + 1] = ta.y; a[4 * q + 2] = ta.z; a[4 * q + 3] = ta.w;
        b[4 * q] = tb.x; b[4 * q + 1] = tb.y; b[4 * q + 2] = tb.z; b[4 * q + 3] = tb.w;
    }
#pragma unroll
    for (int k = 0; k < 4 * NLD; ++k) o[k] = 0.f;
#pragma unroll
    for (int k = 0; k < D; ++k) { o[2 * k] = -a[k]; o[2 * k + 1] = -b[k]; }
    o[2 * D] = __fmul_rn(a[D], sc);
    o[2 * D + 1] = __fmul_rn(b[D], sc);
#pragma unroll
    for (int q = 0; q < NLD; ++q) recP[pr * NLD + q] = make_float4(o[4 * q], o[4 * q + 1], o[4 * q + 2], o[4 * q + 3]);
}

struct TCParams {
    const float *rec;        // pooled records [npad][F]
    const float4 *recP;      // pair records [npad / 2][NLD] (k_pair_records)
    const uint32_t *maskT;   // labels [npad][words_total], this launch uses words [word0, word0 + 16)
    int words_total;
    int word0;
    const Unit *units;
    int nunits;
    float sc256;             // 256 sc: Psi_ij = w_j psi_ij is quantised to v = floor(sc Psi + 1/2) (15 bits); applied in recP
    float magic;             // kMagicUnsigned, or kMagicSigned when weights can be negative
    uint32_t hixor;          // 0, or 0x80808080 with kMagicSigned: hi digit = 2 byte2 - 128
    uint32_t idesc_hi;       // hi digit: s8 when weights can be negative, else u8
    int nq;                  // 256-column accumulators in use: 2, or 1 when this launch has <= 256 label columns
    void *partial;           // [gridDim.x][GEO::kProducerWarps][GEO::kEpiGroups][32 lanes][2] of Acc
    const uint32_t *bitmap;  // SKIP: bit kb of word row I = K block kb can hold a non-zero quantised Psi for row tile I (k_tile_bitmap)
    int bm_words;            // words per row tile
};

// SKIP: the K blocks of a unit that the bitmap marks, in ascending order -- every role of k_perm_tc walks the same list
// (a unit without a marked block is skipped by every role, barriers and phases untouched).
__device__ __forceinline__ int next_kb(const uint32_t *__restrict__ bmI, int kb, int end)
{
    while (kb < end) {
        const uint32_t w = __ldg(bmI + (kb >> 5)) >> (kb & 31);
        if (w) {
            kb += __ffs((int)w) - 1;
            return kb < end ? kb : end;
        }
        kb = (kb | 31) + 1;
    }
    return end;
}

// One launch = 512 label columns.  Grid: persistent, one CTA per SM, clusters of 2 (an SM pair); unit u is processed
// by cluster u % (gridDim.x / 2).  CTA rank r of the pair owns rows 256 I + 128 r .. + 127 (its psi tile, its half of
// the accumulator rows in its own TMEM) and the label columns [256 q + 128 r, 256 q + 128 r + 128), q = 0, 1.
// WEIGHTED: accumulate w_i Y in double; else exact int64.
template <int D, bool WEIGHTED, class GEO, bool SKIP = false>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(GEO::kThreadsTC, 1) k_perm_tc(TCParams P)
{
    using Acc = typename std::conditional<WEIGHTED, double, long long>::type;
    constexpr int kKB = GEO::kKB, kProducerWarps = GEO::kProducerWarps, kStages = GEO::kStages, kRowsPerThread = GEO::kRowsPerThread;
    constexpr int kEpiGroups = GEO::kEpiGroups, kProducers = GEO::kProducers;
    constexpr int kABytes = GEO::kABytes, kBPlane = GEO::kBPlane, kStageBytes = GEO::kStageBytes;
    constexpr int F = rec_floats(D);
    constexpr int NLD = pair_rec_f4(D);     // 16-byte loads per j pair: float2 (-u_j0k, -u_j1k) k < D, then (s_j0, s_j1)
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    // 1024-byte alignment of the operand tiles (SWIZZLE_128B atoms), keeping the pointer in the shared state space
    uint8_t *smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    // one array, so that the hot loop addresses every barrier as bar0 + constant + 8 * index
    constexpr int kRecSlots = GEO::rec_slots(D);
    __shared__ __align__(8) uint64_t bars_s[2 * kStages + 2 + 2 * kMaxRecSlots];
    uint64_t *const bar_full = bars_s, *const bar_empty = bars_s + kStages, *const bar_rec = bars_s + 2 * kStages + 2;
    uint64_t *const bar_recfree = bar_rec + kMaxRecSlots;  // record slot consumed by all producer warps of this CTA
    uint64_t &bar_accfull = bars_s[2 * kStages], &bar_accempty = bars_s[2 * kStages + 1];
    constexpr uint32_t kRecSlotBytes = (kKB / 2) * NLD * 16;
    uint8_t *recs = smem + kStages * kStageBytes;  // record ring
    __shared__ uint32_t tmem_base_s;

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const uint32_t rank = cluster_ctarank();
    const int cluster_id = blockIdx.x >> 1, nclusters = gridDim.x >> 1;

    if (tid == 0) {
        // full / accempty are used in the leader only (arrivals from the producer warps of BOTH CTAs);
        // empty / accfull receive one multicast tcgen05.commit arrival in each CTA
        const uint32_t nfull = 2 * (kProducerWarps + (P.nq > 1 ? GEO::kHelperWarps : 0));  // the helpers fill the q = 1 planes
        for (int s = 0; s < kStages; ++s) { mbar_init(&bar_full[s], nfull); mbar_init(&bar_empty[s], 1); }
        mbar_init(&bar_accfull, 1);
        mbar_init(&bar_accempty, 2 * kProducerWarps);
        for (int s = 0; s < kRecSlots; ++s) { mbar_init(&bar_rec[s], 1); mbar_init(&bar_recfree[s], kProducerWarps); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == kProducerWarps) {
        asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(&tmem_base_s)));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;");
    }
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();  // barrier inits of the peer are visible before any remote arrive
    tc_fence_after();
    const uint32_t tmem = tmem_base_s;

    if (warp == kProducerWarps) {
        // =========================================================================== MMA issuer (leader CTA, one lane)
        if (rank == 0 && lane == 0) {
            const uint32_t idesc_lo = umma_idesc_i8(false), idesc_hi = P.idesc_hi;
            uint32_t it = 0, un = 0;
            for (int u = cluster_id; u < P.nunits; u += nclusters) {
                const Unit U = P.units[u];
                const uint32_t *bmI = SKIP ? P.bitmap + (long long)U.I * P.bm_words : nullptr;
                const int kb_first = SKIP ? next_kb(bmI, U.kb_begin, U.kb_end) : U.kb_begin;
                if (SKIP && kb_first >= U.kb_end) continue;      // nothing marked: no role touches this unit
                mbar_wait_cluster(&bar_accempty, (un & 1) ^ 1);  // both epilogues of the previous unit have drained TMEM
                tc_fence_after();
                for (int kb = kb_first; kb < U.kb_end; kb = SKIP ? next_kb(bmI, kb + 1, U.kb_end) : kb + 1, ++it) {
                    const int s = it % kStages;
                    mbar_wait_cluster(&bar_full[s], (it / kStages) & 1);
                    tc_fence_after();
                    const uint32_t a_base = smem_u32(smem + s * kStageBytes);
                    const uint32_t b_base = a_base + kABytes;
#pragma unroll
                    for (int q = 0; q < 2; ++q) {
                        if (q >= P.nq) break;
#pragma unroll
                        for (int d = 0; d < 2; ++d)
#pragma unroll
                            for (int ks = 0; ks < kKB / 32; ++ks) {
                                // A digit tile: K chunks of 32 bytes, each a [128 rows x 32 B] SWIZZLE_32B sub-tile
                                const uint64_t da = umma_desc(a_base + d * (kTM * kKB) + ks * (kTM * 32), 16, 256, 6);
                                const uint64_t db = umma_desc(b_base + (q * 2 + d) * kBPlane + ks * 4 * 1024, kBPlane, 1024, 2);
                                const uint32_t acc = (kb > kb_first || d > 0 || ks > 0) ? 1u : 0u;
                                umma_i8_pair(tmem + q * 256, da, db, d == 0 ? idesc_hi : idesc_lo, acc);
                            }
                    }
                    umma_commit_pair(&bar_empty[s]);  // frees the stage in both CTAs when these MMAs have read it
                }
                umma_commit_pair(&bar_accfull);
                ++un;
            }
        }
    } else if (warp == kProducerWarps + 1) {
        // =========================================================================== record loader (each CTA, one lane)
        // The pair records of K block `it` go to ring slot it % kRecSlots by one bulk copy, up to kRecSlots blocks ahead
        // of the producers.  The slot was last read for block it - kRecSlots; every producer warp arrives on the slot's
        // own "consumed" barrier after its last load of it, so the awaited phase (use number it / kRecSlots - 1) can
        // only be followed by the phase that this loader itself enables: no parity aliasing.
        if (lane == 0) {
            uint32_t it = 0;
            for (int u = cluster_id; u < P.nunits; u += nclusters) {
                const Unit U = P.units[u];
                const uint32_t *bmI = SKIP ? P.bitmap + (long long)U.I * P.bm_words : nullptr;
                for (int kb = SKIP ? next_kb(bmI, U.kb_begin, U.kb_end) : U.kb_begin; kb < U.kb_end;
                     kb = SKIP ? next_kb(bmI, kb + 1, U.kb_end) : kb + 1, ++it) {
                    const uint32_t slot = it & (kRecSlots - 1);
                    if (it >= kRecSlots) mbar_wait(&bar_recfree[slot], ((it / kRecSlots) - 1) & 1);
                    bulk_g2s(smem_u32(recs + slot * kRecSlotBytes), P.recP + (long long)kb * (kKB / 2) * NLD, kRecSlotBytes, &bar_rec[slot]);
                }
            }
        }
    } else if (warp < kProducerWarps) {
        // =========================================================================== producers + epilogue
        // psi task of a thread: octet oct of the K block (8 j), rows m_r = mrow0 + 16 r, r < R = 4.  A half-warp holds
        // 8 rows x 2 octets, so its 8-byte A-tile stores fall into 16 different bank pairs (no conflicts).
        constexpr int R = kRowsPerThread, G = kEpiGroups;
        const int og = (lane >> 3) & 1, l8 = lane & 7;
        constexpr int OW = kKB / 16;                 // warps along j (two octets each)
        const int oct = 2 * (warp % OW) + og;
        const int mrow0 = 16 * R * (warp / OW) + 8 * (lane >> 4) + l8;
        const int grp0 = GEO::epi_first(warp >> 2), ngrp = GEO::epi_first((warp >> 2) + 1) - grp0;  // this warp's column groups in the epilogue
        const int lane_base = 32 * (warp & 3);       // TMEM lanes this warp may access
        Acc accQ[G], accR[G];
#pragma unroll
        for (int g = 0; g < G; ++g) { accQ[g] = 0; accR[g] = 0; }
        // Thread constants of the main loop.  They are made opaque to the compiler (keep()), which otherwise
        // rematerialises them from the lane index in every K block to save registers (~45 instructions, profiles/r01c).
        const uint32_t fmask = __float_as_uint(P.magic);  // a masked element: v = 0
        const float magic1 = keep(P.magic + 128.f);        // + half a step: round to nearest
        const float2 magicA = make_float2(magic1, magic1);
        static_assert(kKB * 8 == 2 * kProducers, "a producer thread expands two label words (one per column half q) per K block");
        const int jw = warp;                            // label task: 8 j of the K block, both column halves
        const int jj = 8 * jw + (lane >> 2);            // j (local) of this thread's label words
        const int l3 = lane & 3;
        // byte offsets inside a stage of this thread's stores: A tile (row mrow0, octet oct: K chunk oct >> 2, a
        // [128 rows x 32 B] SWIZZLE_32B sub-tile of 4 KB; row mrow0 + 16 r is 512 r further) and B tile (j = jj, hi plane
        // of column half 0, 16-byte chunk 2 l3 of the 128-column row; SWIZZLE_128B; chunk 2 l3 + 1 is at address ^ 16,
        // the lo plane kBPlane further, column half 1 another 2 kBPlane)
        const int offA = (oct >> 2) * (kTM * 32) + (mrow0 >> 3) * 256 + (mrow0 & 7) * 32 + (((((oct & 3) >> 1) ^ ((mrow0 >> 2) & 1))) << 4) + ((oct & 1) << 3);
        const int offB = kABytes + jw * 1024 + (lane >> 2) * 128 + (((2 * l3) ^ (lane >> 2)) << 4);
        const int offJ = kStages * kStageBytes + 4 * oct * NLD * 16;  // its four j pairs inside a record slot
        // running shared-memory addresses of the current stage / record slot (advanced and wrapped every K block)
        const uint32_t bar0 = smem_u32(bars_s);
        uint32_t paA = smem_u32(smem) + offA, pbB = smem_u32(smem) + offB, pjJ = smem_u32(smem) + offJ;
        uint32_t it = 0, un = 0, st = 0, pe = 0;   // K blocks done, units done, stage index it % kStages, its phase (it / kStages) & 1
        for (int u = cluster_id; u < P.nunits; u += nclusters) {
            const Unit U = P.units[u];
            const uint32_t *bmI = SKIP ? P.bitmap + (long long)U.I * P.bm_words : nullptr;
            const int kb_first = SKIP ? next_kb(bmI, U.kb_begin, U.kb_end) : U.kb_begin;
            if (SKIP && kb_first >= U.kb_end) continue;      // nothing marked: no role touches this unit
            const int row0 = U.I * kTM2 + (int)rank * kTM;   // npad < 2^31
            // this thread's i rows; the packed FP32 instructions take (u_ik, u_ik) as a scalar-broadcast operand (R.F32 in SASS)
            float2 ui2[R][D];
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const float4 *p = reinterpret_cast<const float4 *>(P.rec + (long long)(row0 + mrow0 + 16 * r) * F);
                float v[F];
#pragma unroll
                for (int qq = 0; qq < F / 4; ++qq) {
                    const float4 t = __ldg(p + qq);
                    v[4 * qq] = t.x; v[4 * qq + 1] = t.y; v[4 * qq + 2] = t.z; v[4 * qq + 3] = t.w;
                }
                // one register per coordinate (a materialised pair cost 20 registers at D = 5: config 4 -0.9 %, dim 6-8 -8..10 %)
#pragma unroll
                for (int k = 0; k < D; ++k) ui2[r][k] = make_float2(v[k], v[k]);
            }
            // K blocks below kb_diag overlap (or lie below) the rows of this CTA: there only j > i is kept, i.e. element
            // (r, t) of this thread's tile is dropped when kb * kKB + t <= dthr + 16 r
            const int kb_diag = (row0 + kTM + kKB - 1) / kKB;
            const int dthr = row0 + mrow0 - 8 * oct;
            // this thread's label words of K block kb, prefetched one block ahead into registers.  The element index is
            // 64 bits wide: npadK * words_total passes 2^32 at 2 M pooled rows with the maximum permutation count.
            // (the word of the second accumulator, q = 1, is expanded by the helper warps)
            unsigned long long im = (unsigned long long)(kb_first * kKB + jj) * (unsigned)P.words_total + (unsigned)(P.word0 + 4 * (int)rank + l3);
            uint32_t mw = __ldg(P.maskT + im);
            int kb_next = 0;
            for (int kb = kb_first; kb < U.kb_end; kb = kb_next, ++it) {
                const uint32_t mcur = mw;
                kb_next = SKIP ? next_kb(bmI, kb + 1, U.kb_end) : kb + 1;
                if (kb_next < U.kb_end) {
                    im += (unsigned long long)(unsigned)((kb_next - kb) * kKB) * (unsigned)P.words_total;
                    mw = __ldg(P.maskT + im);
                }
                mbar_wait_a(bar0 + 8 * (2 * kStages + 2) + 8 * (it & (kRecSlots - 1)), (it / kRecSlots) & 1);
                mbar_wait_a(bar0 + 8 * kStages + 8 * st, pe ^ 1);

                // ---- psi tile: rows mrow0 + 16 r, j = 8 oct .. 8 oct + 7; label tile: j = jj, this CTA's word
                //      8 q + 4 rank + l3 -> 32 columns, byte p of a word is label bit beta(p): register t of the lo plane is
                //      (m >> t) & 0x01010101 (bytes a), of the hi plane (m << (7 - t)) & 0x80808080 (bytes 128 a).
                //      The four 16-byte label stores are issued between the four j pairs of the psi tile, so that the ALU-pipe
                //      work of the expansion overlaps the FMA-pipe work of the distances (round 1, profiles/r01g_README.md history).
                const uint32_t pbB1 = pbB ^ 16u;  // stage bases are 1024-byte aligned
                auto tile = [&](auto diag_tag) {
                    constexpr bool DIAG = decltype(diag_tag)::value;
                    const int x = kb * kKB - dthr;  // DIAG: element (r, t) is dropped when x <= 16 r - t
                    uint32_t pk[R][4];              // bytes 1 and 2 of (f_2tp, f_2tp+1): (lo, lo, v >> 8, v >> 8) of two j
#pragma unroll
                    for (int tp = 0; tp < 4; ++tp) {
                        float2 nu[2 * NLD];
#pragma unroll
                        for (int qq = 0; qq < NLD; ++qq) {
                            const float4 v = lds128(pjJ + (tp * NLD + qq) * 16);
                            nu[2 * qq] = make_float2(v.x, v.y);
                            nu[2 * qq + 1] = make_float2(v.z, v.w);
                        }
                        {
                            uint32_t q[4];
                            if (tp < 2) {
#pragma unroll
                                for (int t = 0; t < 4; ++t) q[t] = (mcur >> (4 * tp + t)) & 0x01010101u;
                                sts128((tp == 0 ? pbB : pbB1) + kBPlane, make_uint4(q[0], q[1], q[2], q[3]));
                            } else {
#pragma unroll
                                for (int t = 0; t < 4; ++t) q[t] = (mcur << (7 - (4 * (tp - 2) + t))) & 0x80808080u;
                                sts128(tp == 2 ? pbB : pbB1, make_uint4(q[0], q[1], q[2], q[3]));
                            }
                        }
                        {
#pragma unroll
                            for (int r = 0; r < R; ++r) {
                                float2 dd = __fadd2_rn(ui2[r][0], nu[0]);
                                float2 e = __fmul2_rn(dd, dd);
#pragma unroll
                                for (int k = 1; k < D; ++k) {
                                    dd = __fadd2_rn(ui2[r][k], nu[k]);
                                    e = __ffma2_rn(dd, dd, e);
                                }
                                const float2 f2 = __ffma2_rz(make_float2(ex2_approx(-e.x), ex2_approx(-e.y)), nu[D], magicA);
                                uint32_t f0 = __float_as_uint(f2.x), f1 = __float_as_uint(f2.y);
                                if (DIAG) {
                                    if (x <= 16 * r - 2 * tp) f0 = fmask;
                                    if (x <= 16 * r - 2 * tp - 1) f1 = fmask;
                                }
                                pk[r][tp] = __byte_perm(f0, f1, 0x6251);
                            }
                        }
                    }
                    {
#pragma unroll
                        for (int r = 0; r < R; ++r) {
                            uint2 lo, hi;
                            lo.x = __byte_perm(pk[r][0], pk[r][1], 0x5410);
                            lo.y = __byte_perm(pk[r][2], pk[r][3], 0x5410);
                            hi.x = __byte_perm(pk[r][0], pk[r][1], 0x7632);
                            hi.y = __byte_perm(pk[r][2], pk[r][3], 0x7632);
                            // hi digit = 2 (v >> 8) per byte: every byte2 is <= 127, so the word add has no carries
                            // between bytes; with signed weights byte2 = 64 + (v >> 8) and 2 byte2 - 128 = 2 byte2 ^ 0x80
                            hi.x += hi.x;
                            hi.y += hi.y;
                            if (WEIGHTED) { hi.x ^= P.hixor; hi.y ^= P.hixor; }
                            // row m = mrow0 + 16 r: 8-row group m >> 3 advances by 2 (512 bytes), the swizzle phase is that of mrow0
                            sts64(paA + 512 * r, hi);
                            sts64(paA + kTM * kKB + 512 * r, lo);
                        }
                    }
                };
                if (kb < kb_diag) tile(std::true_type{});   // K block overlaps (or lies below) the rows of this CTA: keep only j > i
                else tile(std::false_type{});
                fence_async_smem();
                __syncwarp();
                if (lane == 0) {
                    mbar_arrive_cluster(mapa_rank(bar0 + 8 * st, 0));
                    mbar_arrive(&bar_recfree[it & (kRecSlots - 1)]);  // this warp has read the block's records
                }
                const bool wrapS = st == kStages - 1, wrapJ = ((it + 1) & (kRecSlots - 1)) == 0;
                st = wrapS ? 0 : st + 1;
                pe ^= wrapS ? 1u : 0u;
                paA += wrapS ? (uint32_t)(kStageBytes - kStages * kStageBytes) : (uint32_t)kStageBytes;
                pbB += wrapS ? (uint32_t)(kStageBytes - kStages * kStageBytes) : (uint32_t)kStageBytes;
                pjJ += wrapJ ? kRecSlotBytes - kRecSlots * kRecSlotBytes : kRecSlotBytes;
            }
            // ---- epilogue of the unit: this CTA's 128 rows x 512 columns -------------------------------------
            mbar_wait(&bar_accfull, un & 1);
            tc_fence_after();
            {
                const long long row = (long long)row0 + lane_base + lane;
                const uint32_t *mp = P.maskT + row * P.words_total + P.word0;
                const uint32_t w0 = __ldg(mp);
                const bool real = (w0 >> 2) & 1u;
                const float wf = P.rec[row * F + D];
                const uint32_t taddr = tmem + ((uint32_t)lane_base << 16);
                const int yones = (int)tmem_ld1(taddr + 8);  // label column 2 (all ones) is byte beta^-1(2) = 8 of word 0
                Acc wi, zi;
                if (WEIGHTED) { wi = (Acc)wf; zi = wi * (Acc)yones; }
                else { wi = 1; zi = (Acc)yones; }
#pragma unroll 1
                for (int g = 0; g < ngrp; ++g) {
                    if (grp0 + g >= 8 * P.nq) break;  // one accumulator in use: columns 256.. were never written
                    const uint32_t mword = __ldg(mp + grp0 + g);
                    uint32_t v[32];
                    tmem_ld32(taddr + 32 * (grp0 + g), v);
                    Acc x[32];
#pragma unroll
                    for (int b = 0; b < 32; ++b) x[b] = ((mword >> beta(b)) & 1u) ? wi * (Acc)(int)v[b] : (Acc)0;
                    const Acc qs = lane_transpose_sum(x, lane);
#pragma unroll
                    for (int b = 0; b < 32; ++b) x[b] = (real ? wi * (Acc)(int)v[b] : (Acc)0) + (((mword >> beta(b)) & 1u) ? zi : (Acc)0);
                    const Acc rs = lane_transpose_sum(x, lane);
#pragma unroll
                    for (int gg = 0; gg < G; ++gg)
                        if (gg == g) { accQ[gg] += qs; accR[gg] += rs; }
                }
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive_cluster(mapa_rank(smem_u32(&bar_accempty), 0));
            ++un;
        }
        // per-warp partial column sums: partial[cta][warp][g][lane][2]; lane L of group g = TMEM column 32 (grp0 + g) + L
        Acc *out = reinterpret_cast<Acc *>(P.partial) + ((long long)blockIdx.x * kProducerWarps + warp) * G * 32 * 2;
#pragma unroll
        for (int g = 0; g < G; ++g) {
            out[(g * 32 + lane) * 2] = accQ[g];
            out[(g * 32 + lane) * 2 + 1] = accR[g];
        }
    } else if (P.nq > 1) {
        // =========================================================================== label helpers (second accumulator)
        // The two helper warps expand the label words of the column half q = 1 (word 8 + 4 rank + l3 of every j of the K
        // block) into the q = 1 planes of the B tile, so that a producer thread expands one word per K block instead of
        // two.  They cost no registers (18 warps are allocated as 20, 14 as 16) and take about a tenth of the producers'
        // instructions; the "full" barrier counts their arrivals too.  Lane -> (l3 = lane & 3, j = 8 (NW h + i) + (lane >> 2)),
        // i < NW = kKB / 16: the same (j, 16-byte chunk) -> address map as the producers' label stores.
        constexpr int NW = kKB / (8 * GEO::kHelperWarps);
        const int h = warp - (kProducerWarps + 2), l3 = lane & 3, jsub = lane >> 2;
        const uint32_t bar0 = smem_u32(bars_s);
        uint32_t pbB = smem_u32(smem) + kABytes + (NW * h) * 1024 + jsub * 128 + (((2 * l3) ^ jsub) << 4);
        uint32_t st = 0, pe = 0;
        const unsigned long long jstride = 8ull * (unsigned)P.words_total;
        for (int u = cluster_id; u < P.nunits; u += nclusters) {
            const Unit U = P.units[u];
            const uint32_t *bmI = SKIP ? P.bitmap + (long long)U.I * P.bm_words : nullptr;
            const int kb_first = SKIP ? next_kb(bmI, U.kb_begin, U.kb_end) : U.kb_begin;
            unsigned long long im = (unsigned long long)(kb_first * kKB + 8 * NW * h + jsub) * (unsigned)P.words_total +
                                    (unsigned)(P.word0 + 8 + 4 * (int)rank + l3);
            uint32_t mw[NW];
            if (kb_first < U.kb_end) {
#pragma unroll
                for (int i = 0; i < NW; ++i) mw[i] = __ldg(P.maskT + im + i * jstride);
            }
            int kb_next = 0;
            for (int kb = kb_first; kb < U.kb_end; kb = kb_next) {
                uint32_t cur[NW];
#pragma unroll
                for (int i = 0; i < NW; ++i) cur[i] = mw[i];
                kb_next = SKIP ? next_kb(bmI, kb + 1, U.kb_end) : kb + 1;
                if (kb_next < U.kb_end) {
                    im += (unsigned long long)(unsigned)((kb_next - kb) * kKB) * (unsigned)P.words_total;
#pragma unroll
                    for (int i = 0; i < NW; ++i) mw[i] = __ldg(P.maskT + im + i * jstride);
                }
                mbar_wait_a(bar0 + 8 * kStages + 8 * st, pe ^ 1);   // the stage is free
#pragma unroll
                for (int i = 0; i < NW; ++i) {
                    const uint32_t b0 = pbB + i * 1024, b1 = b0 ^ 16u, m = cur[i];
                    uint32_t q[4];
#pragma unroll
                    for (int t = 0; t < 4; ++t) q[t] = (m >> t) & 0x01010101u;
                    sts128(b0 + 3 * kBPlane, make_uint4(q[0], q[1], q[2], q[3]));
#pragma unroll
                    for (int t = 0; t < 4; ++t) q[t] = (m >> (4 + t)) & 0x01010101u;
                    sts128(b1 + 3 * kBPlane, make_uint4(q[0], q[1], q[2], q[3]));
#pragma unroll
                    for (int t = 0; t < 4; ++t) q[t] = (m << (7 - t)) & 0x80808080u;
                    sts128(b0 + 2 * kBPlane, make_uint4(q[0], q[1], q[2], q[3]));
#pragma unroll
                    for (int t = 0; t < 4; ++t) q[t] = (m << (3 - t)) & 0x80808080u;
                    sts128(b1 + 2 * kBPlane, make_uint4(q[0], q[1], q[2], q[3]));
                }
                fence_async_smem();
                __syncwarp();
                if (lane == 0) mbar_arrive_cluster(mapa_rank(bar0 + 8 * st, 0));
                const bool wrapS = st == kStages - 1;
                st = wrapS ? 0 : st + 1;
                pe ^= wrapS ? 1u : 0u;
                pbB += wrapS ? (uint32_t)(kStageBytes - kStages * kStageBytes) : (uint32_t)kStageBytes;
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();  // the peer may still be reading this CTA's shared memory / TMEM through the pair's MMAs
    if (warp == kProducerWarps) asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, 512;" ::"r"(tmem));
}

// Column sums over CTAs and warps, fixed order: TMEM column 32 gc + lane (gc = c >> 5) is held by the four warps
// 4 (gc / G) .. + 3 as their group gc % G, and is label column c = 32 gc + beta(lane).  raw[col] = Q, raw[512 + col] = R
// as exact integers (or doubles when weighted) in units of the quantisation step: what a unit-range shard exchanges.
template <bool WEIGHTED, class GEO>
__global__ void k_tc_reduce(const void *partial, int ncta, void *raw)
{
    using Acc = typename std::conditional<WEIGHTED, double, long long>::type;
    constexpr int kEpiWarps = GEO::kEpiWarps, kEpiGroups = GEO::kEpiGroups, kProducerWarps = GEO::kProducerWarps;
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= kCols) return;
    constexpr int G = kEpiGroups;
    const int gc = c >> 5, lane = c & 31;
    int e = 0;  // warp row that reads column group gc in the epilogue
    while (e + 1 < kEpiWarps && GEO::epi_first(e + 1) <= gc) ++e;
    const int g = gc - GEO::epi_first(e);
    const Acc *p = reinterpret_cast<const Acc *>(partial);
    Acc sq = 0, sr = 0;
    for (int b = 0; b < ncta; ++b)
        for (int w = 4 * e; w < 4 * e + 4; ++w) {
            const Acc *e = p + (((long long)b * kProducerWarps + w) * G * 32 + g * 32 + lane) * 2;
            sq += e[0];
            sr += e[1];
        }
    const int col = (c & ~31) + beta(lane);
    reinterpret_cast<Acc *>(raw)[col] = sq;
    reinterpret_cast<Acc *>(raw)[kCols + col] = sr;
}
// out[c] = {Q, R} as doubles in units of psi (divided by sc)
template <bool WEIGHTED>
__global__ void k_tc_scale(const void *raw, double inv_sc, double *__restrict__ outQ, double *__restrict__ outR)
{
    using Acc = typename std::conditional<WEIGHTED, double, long long>::type;
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= kCols) return;
    outQ[c] = (double)reinterpret_cast<const Acc *>(raw)[c] * inv_sc;
    outR[c] = (double)reinterpret_cast<const Acc *>(raw)[kCols + c] * inv_sc;
}

// Label words of the TC layout: maskT[pos][chunk * 16 + W], column c = 32 W + b of chunk ch:
// c = 0 observed (pooled index < n_x), c = 1 second labelling (class segment of i in `lab2_classes`), c = 2 ones,
// c >= 3 permutation p = ch * 509 + c - 3 (local index; global p0 + p) if p < nperm.  grid = (events, chunks * 16).
__global__ void __launch_bounds__(kThreads) k_label_write_tc(long long N, long long n_x, int nperm, long long p0, uint32_t seed_lo,
                                                            uint32_t seed_hi, const SelState *__restrict__ st, LabelOut L,
                                                            unsigned lab2_classes, int words_total, const int *__restrict__ inv,
                                                            uint32_t *__restrict__ maskT)
{
    const long long i = blockIdx.x * (long long)kThreads + threadIdx.x;
    const int ch = blockIdx.y / kWordsPerChunk, W = blockIdx.y % kWordsPerChunk;
    if (i >= N) return;
    long long pos = i;
    int cls = 0;
    for (int s = 0; s < L.nseg; ++s)
        if (i >= L.seg_first[s] && i < L.seg_first[s + 1]) { pos = L.seg_pos[s] + (i - L.seg_first[s]); cls = s; }
    uint32_t word = 0u;
    uint64_t K[4];
    long long have_p4 = -1;
    for (int b = 0; b < 32; ++b) {
        const int c = 32 * W + b;
        if (c == 0) { if (i < n_x) word |= 1u; continue; }
        if (c == 1) { if ((lab2_classes >> cls) & 1u) word |= 2u; continue; }
        if (c == 2) { word |= 4u; continue; }
        const int p = ch * kPermsPerChunk + c - kSpecial;
        if (p >= nperm) break;
        const long long pg = p0 + p;
        if ((pg >> 2) != have_p4) { have_p4 = pg >> 2; label_keys4((uint32_t)i, (uint32_t)have_p4, seed_lo, seed_hi, K); }
        if (K[pg & 3] <= st[p].prefix) word |= 1u << b;
    }
    if (inv) pos = inv[pos];  // row of the contraction's own order (k_morton_keys)
    maskT[pos * words_total + blockIdx.y] = word;
}

// ---- row order of the contraction -----------------------------------------------------------------------------------
// The sums of k_perm_tc do not depend on the order of the rows inside a class segment (unit weights: bit for bit, every
// pair enters once with a symmetric quantised psi), but its TIME does: the board runs at its power cap and the energy of
// an MMA follows the operand bits -- with neighbouring rows close in phase space the digit tiles of neighbouring j are
// alike and far tiles are mostly zero: -2.3 % per launch at config 4 (profiles/r02_README.md).  So the contraction
// runs on a copy of the records in Morton order: key = class << 20 | interleaved bits of the coordinates quantised over the
// bounding box (written by k_prep from the input coordinates; padding rows: the largest key of their class, so every class
// keeps its row range), a stable radix sort of
// (key, row) (k_rs_*: two passes of 11 bits over the 22-bit key), then order[new] = old, inv[old] = new and recS[new] = rec[old].  The labels are written through inv; the
// escalation and every other kernel keep the layout order.
// the keys come from k_prep (PrepParams::key); the sort works on a copy and starts from the identity order
__global__ void __launch_bounds__(kThreads) k_key_iota(const uint32_t *__restrict__ key_in, long long npad, uint32_t *__restrict__ key, int *__restrict__ idx)
{
    const long long row = blockIdx.x * (long long)kThreads + threadIdx.x;
    if (row >= npad) return;
    key[row] = key_in[row];
    idx[row] = (int)row;
}
// Stable LSD radix sort of (key, value) pairs, kRsBits bits per pass: one warp per tile of `tile` consecutive elements
// (a multiple of 32).  k_rs_hist: hist[bin * ntiles + t] = elements of tile t in bin; k_rs_scan: exclusive prefix in place
// (bin-major, so equal digits keep their tile order); k_rs_scatter: the rank of an element inside its tile is the count of
// earlier elements with the same digit -- earlier steps from the warp's shared-memory counter, the same step from
// __match_any_sync -- so the pass is stable.
constexpr int kRsBits = 11, kRsBins = 1 << kRsBits, kRsWarps = 4;
__global__ void __launch_bounds__(32 * kRsWarps) k_rs_hist(const uint32_t *__restrict__ key, long long n, int shift, long long tile, long long ntiles,
                                                          uint32_t *__restrict__ hist)
{
    __shared__ uint32_t cnt[kRsWarps][kRsBins];
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const long long t = blockIdx.x * (long long)kRsWarps + w;
    for (int b = lane; b < kRsBins; b += 32) cnt[w][b] = 0u;
    __syncwarp();
    if (t < ntiles) {
        for (long long i = t * tile + lane; i < min(n, (t + 1) * tile); i += 32) atomicAdd(&cnt[w][(key[i] >> shift) & (kRsBins - 1)], 1u);
        __syncwarp();
        for (int b = lane; b < kRsBins; b += 32) hist[(long long)b * ntiles + t] = cnt[w][b];
    }
}
// exclusive prefix sum of `total` counters in place; one block of 1024 threads, a contiguous chunk per thread
__global__ void __launch_bounds__(1024) k_rs_scan(uint32_t *__restrict__ hist, long long total)
{
    __shared__ uint32_t part[1024];
    const long long chunk = (total + 1023) / 1024, a = threadIdx.x * chunk, b = min(total, a + chunk);
    uint32_t sum = 0u;
    for (long long i = a; i < b; ++i) sum += hist[i];
    part[threadIdx.x] = sum;
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t run = 0u;
        for (int k = 0; k < 1024; ++k) { const uint32_t v = part[k]; part[k] = run; run += v; }
    }
    __syncthreads();
    uint32_t run = part[threadIdx.x];
    for (long long i = a; i < b; ++i) { const uint32_t v = hist[i]; hist[i] = run; run += v; }
}
__global__ void __launch_bounds__(32 * kRsWarps) k_rs_scatter(const uint32_t *__restrict__ key_in, const int *__restrict__ val_in, long long n, int shift,
                                                             long long tile, long long ntiles, const uint32_t *__restrict__ off,
                                                             uint32_t *__restrict__ key_out, int *__restrict__ val_out)
{
    __shared__ uint32_t cnt[kRsWarps][kRsBins];
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const long long t = blockIdx.x * (long long)kRsWarps + w;
    for (int b = lane; b < kRsBins; b += 32) cnt[w][b] = 0u;
    __syncwarp();
    if (t >= ntiles) return;
    const long long end = min(n, (t + 1) * tile);
    for (long long i0 = t * tile; i0 < end; i0 += 32) {   // tile is a multiple of 32: the trip count is the warp's
        const long long i = i0 + lane;
        const bool valid = i < end;
        const uint32_t k = valid ? key_in[i] : 0u;
        const uint32_t d = valid ? (k >> shift) & (kRsBins - 1) : (uint32_t)kRsBins;   // invalid lanes: a group of their own
        const unsigned peers = __match_any_sync(0xffffffffu, d);
        const uint32_t base = valid ? cnt[w][d] : 0u;
        __syncwarp();
        if (valid && lane == __ffs((int)peers) - 1) cnt[w][d] = base + (uint32_t)__popc(peers);
        __syncwarp();
        if (valid) {
            const long long pos = (long long)off[(long long)d * ntiles + t] + base + (uint32_t)__popc(peers & ((1u << lane) - 1u));
            key_out[pos] = k;
            val_out[pos] = val_in[i];
        }
    }
}

// inv[order[r]] = r, recS[r] = rec[order[r]] (F4 float4 per row); one thread per float4
__global__ void k_order_gather(const float4 *__restrict__ rec, const int *__restrict__ order, long long npad, int F4, int *__restrict__ inv,
                               float4 *__restrict__ recS)
{
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < npad * F4; k += (long long)gridDim.x * blockDim.x) {
        const long long r = k / F4;
        const int q = (int)(k % F4), old = order[r];
        if (q == 0) inv[old] = (int)r;
        recS[k] = rec[(long long)old * F4 + q];
    }
}

// ---- exact skipping of far K blocks (SKIP) -------------------------------------------------------------------------
// v = floor(sc Psi + 1/2) is 0 for every pair with |u_i - u_j|^2 > log2(2 sc) = 16.0 (unit weights), i.e. farther apart than
// 4.7 sigma: a (row tile, K block) pair whose bounding boxes are farther apart than that contributes exactly nothing to
// any integer sum and is not evaluated at all -- no psi, no labels, no MMAs; the sums stay the same bits.  It pays where
// the sample is wide in units of sigma and the rows are in Morton order (the Dalitz plot at sigma = 0.1: 59 % of the K
// blocks); run_perm_tc_g takes the SKIP kernel only when the bitmap marks less than 95 % of the blocks.
// Bounding boxes of consecutive groups of `rows_per_box` rows (real rows only: weight != 0); one warp per box.
constexpr float kSkipDist2 = 16.1f;  // > log2(65532) = 15.99998 with room for the fp32 rounding of the distance and of ex2.approx
__global__ void __launch_bounds__(kThreads) k_row_boxes(const float *__restrict__ rec, int F, int dim, long long nrows, int rows_per_box,
                                                       long long nboxes, float *__restrict__ lo, float *__restrict__ hi)
{
    const long long box = blockIdx.x * (long long)(kThreads / 32) + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (box >= nboxes) return;
    float a[kMaxDimTC], b[kMaxDimTC];
#pragma unroll
    for (int k = 0; k < kMaxDimTC; ++k) { a[k] = 3.0e38f; b[k] = -3.0e38f; }
    for (int r = lane; r < rows_per_box; r += 32) {
        const long long row = box * rows_per_box + r;
        if (row >= nrows || rec[row * F + dim] == 0.f) continue;
#pragma unroll
        for (int k = 0; k < kMaxDimTC; ++k)
            if (k < dim) { const float v = rec[row * F + k]; a[k] = fminf(a[k], v); b[k] = fmaxf(b[k], v); }
    }
#pragma unroll
    for (int k = 0; k < kMaxDimTC; ++k) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            a[k] = fminf(a[k], __shfl_xor_sync(0xffffffffu, a[k], o));
            b[k] = fmaxf(b[k], __shfl_xor_sync(0xffffffffu, b[k], o));
        }
        if (lane == 0) { lo[box * kMaxDimTC + k] = a[k]; hi[box * kMaxDimTC + k] = b[k]; }
    }
}
// bitmap[I][kb >> 5] bit kb & 31 = the boxes of row tile I and K block kb are within kSkipDist2 (and kb is not below the
// tile's first block); marked += the number of marked blocks.  grid = row tiles, block = kThreads.
__global__ void __launch_bounds__(kThreads) k_tile_bitmap(const float *__restrict__ tlo, const float *__restrict__ thi, const float *__restrict__ klo,
                                                         const float *__restrict__ khi, int dim, int NK, int kKB, int bm_words,
                                                         uint32_t *__restrict__ bitmap, unsigned long long *__restrict__ marked)
{
    const int I = blockIdx.x, lane = threadIdx.x & 31;
    const int kb0 = (int)((long long)I * kTM2 / kKB);
    float a[kMaxDimTC], b[kMaxDimTC];
#pragma unroll
    for (int k = 0; k < kMaxDimTC; ++k) { a[k] = tlo[(long long)I * kMaxDimTC + k]; b[k] = thi[(long long)I * kMaxDimTC + k]; }
    unsigned int cnt = 0;
    for (int kb = threadIdx.x; kb < bm_words * 32; kb += kThreads) {
        bool need = false;
        if (kb >= kb0 && kb < NK) {
            float d2 = 0.f;
#pragma unroll
            for (int k = 0; k < kMaxDimTC; ++k)
                if (k < dim) {
                    const float g = fmaxf(0.f, fmaxf(klo[(long long)kb * kMaxDimTC + k] - b[k], a[k] - khi[(long long)kb * kMaxDimTC + k]));
                    d2 = fmaf(g, g, d2);
                }
            need = d2 <= kSkipDist2;   // an empty box (3e38 / -3e38) gives inf: not needed
        }
        const unsigned int w = __ballot_sync(0xffffffffu, need);
        if (lane == 0) { bitmap[(long long)I * bm_words + (kb >> 5)] = w; cnt += __popc(w); }
    }
    if (lane == 0 && cnt) atomicAdd(marked, (unsigned long long)cnt);
}

// W_c = sum_i a_ic w_i for every column of the TC layout.  grid = (row chunks, words_total); lane = bit.
__global__ void __launch_bounds__(kThreads) k_perm_W_tc(const float *__restrict__ rec, int F, int dim, const uint32_t *__restrict__ maskT,
                                                       int words_total, long long npad, int nchunk, double *__restrict__ partials)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, wd = blockIdx.y;
    const long long rows_per_chunk = (npad + nchunk - 1) / nchunk;
    const long long r0 = blockIdx.x * rows_per_chunk, r1 = min(npad, r0 + rows_per_chunk);
    double W = 0.0;
    for (long long i = r0 + warp; i < r1; i += kThreads / 32) {
        const uint32_t m = maskT[i * words_total + wd];
        if (m >> lane & 1u) W += (double)rec[i * F + dim];
    }
    __shared__ double s[kThreads / 32][32];
    s[warp][lane] = W;
    __syncthreads();
    if (threadIdx.x < 32) {
        double t = 0.0;
#pragma unroll
        for (int w = 0; w < kThreads / 32; ++w) t += s[w][threadIdx.x];
        partials[((long long)wd * nchunk + blockIdx.x) * 32 + threadIdx.x] = t;
    }
}

}  // namespace tc
}  // namespace et
