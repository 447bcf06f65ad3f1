// et_api.cu -- host side of libet.so: context, argument checking, staging, kernel orchestration.
// The C ABI is declared in include/et.h.  Nothing here computes on the CPU beyond O(1) bookkeeping: every step
// of the path (prep, split, labels, all-pairs sums, permutation sums, the statistic and the p-value) is a kernel.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <algorithm>
#include <vector>

#include <nvtx3/nvToolsExt.h>  // header-only NVTX v3: ranges for Nsight tools, a no-op when no tool is attached

#include "../../include/et.h"
#include "et_kernels.cuh"
#include "et_tc.cuh"
#include "et_scp.cuh"

using namespace et;

namespace {

struct Buf {
    void *p = nullptr;
    size_t cap = 0;
};

struct Layout {
    int ncls = 2;
    long long n = 0, nbar = 0, N = 0, npad = 0;
    long long seg_first[kMaxCls + 1] = {0};  // first pooled (label) index of each class segment
    long long seg_count[kMaxCls] = {0};
    long long seg_pos[kMaxCls + 1] = {0};    // first padded row of each class segment
    long long n_a = 0;                       // size of the first sample of the two-sample test (classes < split)
    int split = 1;                           // classes [0, split) form sample A, the rest sample B
};

}  // namespace

struct et_ctx {
    int device = 0;
    int num_sms = 0;
    cudaStream_t stream = nullptr;
    bool own_stream = false;
    char err[512] = {0};
    // scratch (grow-only)
    Buf in_x, in_xbar, in_wx, in_wxbar, in_mx, in_mb, in_aux;
    Buf rec, tilecls, partials, sums, rowsum, mask, sel, hist, partQ, Q, partRW, RW, mm, flag, counter;
    Buf src, posx, posb, blkcnt, totals, clsw, clssum, result, tperm, rows, rowsout, count64;
    void *pinned = nullptr;
    size_t pinned_cap = 0;
    // events / stats
    cudaEvent_t ev[8] = {nullptr};
    et_stats stats = {};
    double acc_pairs_ms = 0, acc_labels_ms = 0;
    // per kernel class (KC_*): device ms, launches and algorithmic ops of the current call
    double kc_ms[4] = {0, 0, 0, 0};
    int64_t kc_launches[4] = {0, 0, 0, 0};
    int64_t kc_ops[4] = {0, 0, 0, 0};
    int64_t opt_perm_kernel = 0;
    int64_t opt_perm_offset = 0;
    int64_t opt_exact_p = 16;       // guard-band escalation: re-evaluate up to this many near permutations (0 = off)
    // unit-range shard (et_set_shard): this context evaluates work units u = shard_rank (mod shard_world) of the O(N^2)
    // kernels and completes the partial sums through the caller's all-gather
    int shard_rank = 0, shard_world = 1;
    et_allgather_fn shard_fn = nullptr;
    void *shard_user = nullptr;
    Buf shardbuf;
    Buf rec2, tilecls2, esccls, escD, nearbuf, escw;
    double wmin = 1.0, wmax = 1.0;  // range of the fp32-rounded weights of the last prep (1, 1 when unweighted)
    double umax2 = 0.0;             // bound of |u|^2 over the records of the last prep: squared half diagonal of the bounding box, scaled
    int64_t opt_distance = 0;       // ET_OPT_DISTANCE
    int64_t opt_label_select = 0;   // ET_OPT_LABEL_SELECT
    Buf maskT, units, tcpart, tcQ, tcR, tcWpart, tcW, recP, tcraw;
    Buf scpcnt, scpS;
    Buf selcand, selsave;  // radix select: candidate lists of the index half, state after the key32 half
    // row order of the tensor-core contraction (et_tc.cuh, k_morton_keys): keys, order[new] = old, inv[old] = new, sorted records
    Buf tckey, tckey2, tcidx, tcorder, tcinv, recS, rshist;  // rshist: the radix sort's histogram
    Buf tcboxes, tcbitmap;          // exact skipping of far K blocks: bounding boxes, bitmap[row tile][K block]
    int64_t opt_tc_skip = 1;        // ET_OPT_TC_SKIP
    bool tc_sorted = false;         // maskT of the last label write is in the sorted order (tcorder / tcinv hold it)
    int64_t opt_tc_order = 1;       // ET_OPT_TC_ORDER
    Buf prepkey;                    // Morton key of every record row (k_prep)
    bool tc_attr_set = false;
    // NVTX ranges: the call and its spans (labels, O(N^2) kernels, escalation); ids of the open ones
    nvtxRangeId_t nvtx_call = 0, nvtx_span[8] = {0};
    bool nvtx_call_open = false, nvtx_span_open[8] = {false};
};

namespace {

enum { KC_T = 0, KC_ROW = 1, KC_PERM32 = 2, KC_PERMTC = 3 };
const char *const kKcName[4] = {"k_pairs_T", "k_pairs_rows", "k_perm32", "k_perm_tc"};

et_status fail(et_ctx *c, et_status st, const char *fmt, ...)
{
    if (c) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(c->err, sizeof(c->err), fmt, ap);
        va_end(ap);
    }
    return st;
}

#define CUDA_TRY(expr)                                                                                   \
    do {                                                                                                 \
        cudaError_t e_ = (expr);                                                                         \
        if (e_ != cudaSuccess)                                                                           \
            return fail(ctx, e_ == cudaErrorMemoryAllocation ? ET_ERR_NOMEM : ET_ERR_CUDA, "%s: %s", #expr, \
                        cudaGetErrorString(e_));                                                         \
    } while (0)
#define ET_TRY(expr)                     \
    do {                                 \
        et_status s_ = (expr);           \
        if (s_ != ET_OK) return s_;      \
    } while (0)

et_status ensure(et_ctx *ctx, Buf &b, size_t bytes)
{
    if (bytes == 0) bytes = 16;
    if (b.cap >= bytes) return ET_OK;
    if (b.p) CUDA_TRY(cudaFree(b.p));
    b.p = nullptr;
    b.cap = 0;
    CUDA_TRY(cudaMalloc(&b.p, bytes));
    b.cap = bytes;
    return ET_OK;
}

et_status ensure_pinned(et_ctx *ctx, size_t bytes)
{
    if (ctx->pinned_cap >= bytes) return ET_OK;
    if (ctx->pinned) CUDA_TRY(cudaFreeHost(ctx->pinned));
    ctx->pinned = nullptr;
    ctx->pinned_cap = 0;
    CUDA_TRY(cudaMallocHost(&ctx->pinned, bytes));
    ctx->pinned_cap = bytes;
    return ET_OK;
}

// Returns a device pointer for an input array: the pointer itself (ET_DEVICE) or a staged copy (ET_HOST).
et_status stage_in(et_ctx *ctx, const void *p, size_t bytes, et_memspace mem, Buf &b, const void **out)
{
    if (!p) { *out = nullptr; return ET_OK; }
    if (mem == ET_DEVICE) { *out = p; return ET_OK; }
    ET_TRY(ensure(ctx, b, bytes));
    CUDA_TRY(cudaMemcpyAsync(b.p, p, bytes, cudaMemcpyHostToDevice, ctx->stream));
    *out = b.p;
    return ET_OK;
}

inline size_t elem_size(et_dtype t) { return t == ET_F32 ? 4 : 8; }

et_status check_common(et_ctx *ctx, const void *x, int64_t n, const void *xbar, int64_t nbar, int dim, et_dtype dtype,
                       et_memspace mem, double sigma)
{
    if (!ctx) return ET_ERR_INVALID;
    if (!x || !xbar) return fail(ctx, ET_ERR_INVALID, "null coordinate pointer");
    if (n < 2 || nbar < 2) return fail(ctx, ET_ERR_INVALID, "n and nbar must be >= 2 (Eq. 2 divides by n(n-1)); got %lld, %lld", (long long)n, (long long)nbar);
    if (n + nbar >= (1ll << 31)) return fail(ctx, ET_ERR_INVALID, "n + nbar must be < 2^31");
    if (dim < 1 || dim > ET_MAX_DIM) return fail(ctx, ET_ERR_INVALID, "dim must be in 1..%d; got %d", ET_MAX_DIM, dim);
    if (dtype != ET_F32 && dtype != ET_F64) return fail(ctx, ET_ERR_INVALID, "bad dtype");
    if (mem != ET_HOST && mem != ET_DEVICE) return fail(ctx, ET_ERR_INVALID, "bad memspace");
    if (!(sigma > 0.0) || !std::isfinite(sigma)) return fail(ctx, ET_ERR_SIGMA, "sigma must be finite and > 0");
    return ET_OK;
}

inline long long round_up(long long v, long long m) { return (v + m - 1) / m * m; }

void layout_two(Layout &L, long long n, long long nbar)
{
    L.ncls = 2;
    L.n = n; L.nbar = nbar; L.N = n + nbar;
    L.seg_count[0] = n; L.seg_count[1] = nbar;
    L.seg_first[0] = 0; L.seg_first[1] = n; L.seg_first[2] = n + nbar;
    L.seg_pos[0] = 0; L.seg_pos[1] = round_up(n, kPad); L.seg_pos[2] = L.seg_pos[1] + round_up(nbar, kPad);
    L.npad = L.seg_pos[2];
    L.split = 1;
    L.n_a = n;
}

void layout_four(Layout &L, long long n, long long nbar, const long long cnt[4])
{
    L.ncls = 4;
    L.n = n; L.nbar = nbar; L.N = n + nbar;
    long long first = 0, pos = 0;
    for (int c = 0; c < 4; ++c) {
        L.seg_count[c] = cnt[c];
        L.seg_first[c] = first;
        L.seg_pos[c] = pos;
        first += cnt[c];
        pos += round_up(cnt[c], kPad);
    }
    L.seg_first[4] = first;
    L.seg_pos[4] = pos;
    L.npad = pos;
    L.split = 2;
    L.n_a = cnt[0] + cnt[1];
}

et_status upload_tile_classes(et_ctx *ctx, const Layout &L, Buf *dst = nullptr)
{
    Buf &b = dst ? *dst : ctx->tilecls;
    const long long nt = L.npad / kPad;
    std::vector<uint8_t> cls((size_t)nt);
    for (int c = 0; c < L.ncls; ++c)
        for (long long t = L.seg_pos[c] / kPad; t < L.seg_pos[c + 1] / kPad; ++t) cls[(size_t)t] = (uint8_t)c;
    ET_TRY(ensure(ctx, b, (size_t)nt));
    CUDA_TRY(cudaMemcpyAsync(b.p, cls.data(), (size_t)nt, cudaMemcpyHostToDevice, ctx->stream));
    CUDA_TRY(cudaStreamSynchronize(ctx->stream));  // cls goes out of scope
    return ET_OK;
}

// ---- call bracketing / stats -----------------------------------------------------------------------------
void nvtx_close_all(et_ctx *ctx)
{
    for (int k = 0; k < 8; ++k)
        if (ctx->nvtx_span_open[k]) { nvtxRangeEnd(ctx->nvtx_span[k]); ctx->nvtx_span_open[k] = false; }
    if (ctx->nvtx_call_open) { nvtxRangeEnd(ctx->nvtx_call); ctx->nvtx_call_open = false; }
}

et_status begin_call(et_ctx *ctx)
{
    nvtx_close_all(ctx);  // a call that returned an error left its ranges open
    ctx->nvtx_call = nvtxRangeStartA("libet call");
    ctx->nvtx_call_open = true;
    ctx->stats = et_stats{};
    ctx->acc_pairs_ms = ctx->acc_labels_ms = 0;
    for (int k = 0; k < 4; ++k) { ctx->kc_ms[k] = 0; ctx->kc_launches[k] = 0; ctx->kc_ops[k] = 0; }
    CUDA_TRY(cudaSetDevice(ctx->device));
    CUDA_TRY(cudaEventRecord(ctx->ev[0], ctx->stream));
    return ET_OK;
}
et_status end_call(et_ctx *ctx)
{
    CUDA_TRY(cudaEventRecord(ctx->ev[1], ctx->stream));
    CUDA_TRY(cudaStreamSynchronize(ctx->stream));
    float ms = 0;
    CUDA_TRY(cudaEventElapsedTime(&ms, ctx->ev[0], ctx->ev[1]));
    ctx->stats.ms_total = ms;
    ctx->stats.ms_pairs = ctx->acc_pairs_ms;
    ctx->stats.ms_labels = ctx->acc_labels_ms;
    int dom = 0;
    for (int k = 1; k < 4; ++k)
        if (ctx->kc_ms[k] > ctx->kc_ms[dom]) dom = k;
    ctx->stats.ms_dominant = ctx->kc_ms[dom];
    ctx->stats.dominant_launches = ctx->kc_launches[dom];
    ctx->stats.dominant_ops = ctx->kc_ops[dom];
    snprintf(ctx->stats.dominant_kernel, sizeof(ctx->stats.dominant_kernel), "%s", ctx->kc_launches[dom] ? kKcName[dom] : "");
    nvtx_close_all(ctx);
    return ET_OK;
}
// Bracket a group of launches with events; the elapsed time is read (after a sync) by span_end.
et_status span_begin(et_ctx *ctx, int slot)
{
    if (ctx->nvtx_span_open[slot]) nvtxRangeEnd(ctx->nvtx_span[slot]);
    ctx->nvtx_span[slot] = nvtxRangeStartA(slot == 4 ? "libet labels" : slot == 6 ? "libet escalation" : "libet pair kernels");
    ctx->nvtx_span_open[slot] = true;
    CUDA_TRY(cudaEventRecord(ctx->ev[slot], ctx->stream));
    return ET_OK;
}
et_status span_end(et_ctx *ctx, int slot, double *acc, int kc = -1, int64_t launches = 0, int64_t ops = 0)
{
    CUDA_TRY(cudaEventRecord(ctx->ev[slot + 1], ctx->stream));
    CUDA_TRY(cudaEventSynchronize(ctx->ev[slot + 1]));
    float ms = 0;
    CUDA_TRY(cudaEventElapsedTime(&ms, ctx->ev[slot], ctx->ev[slot + 1]));
    *acc += ms;
    if (ctx->nvtx_span_open[slot]) { nvtxRangeEnd(ctx->nvtx_span[slot]); ctx->nvtx_span_open[slot] = false; }
    if (kc >= 0) { ctx->kc_ms[kc] += ms; ctx->kc_launches[kc] += launches; ctx->kc_ops[kc] += ops; }
    return ET_OK;
}

#define LAUNCH_CHECK()                          \
    do {                                        \
        ctx->stats.launches += 1;               \
        CUDA_TRY(cudaGetLastError());           \
    } while (0)

// ---- prep ------------------------------------------------------------------------------------------------
template <typename TIn>
et_status run_prep_t(et_ctx *ctx, const TIn *x, const TIn *xbar, const double *wx, const double *wxbar, const int *src,
                     const Layout &L, int dim, double sigma)
{
    ET_TRY(ensure(ctx, ctx->mm, 18 * sizeof(uint32_t)));
    ET_TRY(ensure(ctx, ctx->flag, sizeof(int)));
    ET_TRY(ensure_pinned(ctx, 4096));
    uint32_t *h = static_cast<uint32_t *>(ctx->pinned);
    for (int k = 0; k < 9; ++k) { h[2 * k] = 0xffffffffu; h[2 * k + 1] = 0u; }
    CUDA_TRY(cudaMemcpyAsync(ctx->mm.p, h, 18 * sizeof(uint32_t), cudaMemcpyHostToDevice, ctx->stream));
    CUDA_TRY(cudaMemsetAsync(ctx->flag.p, 0, sizeof(int), ctx->stream));
    const int grid = ctx->num_sms * 4;
    k_minmax<TIn><<<grid, 256, 0, ctx->stream>>>(x, L.n, dim, wx, static_cast<uint32_t *>(ctx->mm.p), static_cast<int *>(ctx->flag.p));
    LAUNCH_CHECK();
    k_minmax<TIn><<<grid, 256, 0, ctx->stream>>>(xbar, L.nbar, dim, wxbar, static_cast<uint32_t *>(ctx->mm.p), static_cast<int *>(ctx->flag.p));
    LAUNCH_CHECK();
    CUDA_TRY(cudaMemcpyAsync(h + 32, ctx->mm.p, 18 * sizeof(uint32_t), cudaMemcpyDeviceToHost, ctx->stream));
    CUDA_TRY(cudaMemcpyAsync(h + 64, ctx->flag.p, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
    CUDA_TRY(cudaStreamSynchronize(ctx->stream));
    if (h[64] != 0) return fail(ctx, ET_ERR_NONFINITE, "NaN or Inf in coordinates or weights");
    ctx->wmin = ctx->wmax = 1.0;
    if (wx) { ctx->wmin = (double)key2f(h[32 + 16]); ctx->wmax = (double)key2f(h[32 + 17]); }

    PrepParams P{};
    for (int k = 0; k < dim; ++k) P.centre[k] = 0.5 * ((double)key2f(h[32 + 2 * k]) + (double)key2f(h[32 + 2 * k + 1]));
    P.scale = std::sqrt(1.4426950408889634074 / (2.0 * sigma * sigma));
    ctx->umax2 = 0.0;
    for (int k = 0; k < dim; ++k) {
        const double half = 0.5 * ((double)key2f(h[32 + 2 * k + 1]) - (double)key2f(h[32 + 2 * k])) * P.scale;
        ctx->umax2 += half * half;
        const double half_x = 0.5 * ((double)key2f(h[32 + 2 * k + 1]) - (double)key2f(h[32 + 2 * k]));
        P.inv_half[k] = half_x > 0.0 ? 1.0 / half_x : 0.0;
    }
    P.n = L.n; P.nbar = L.nbar; P.npad = L.npad; P.dim = dim; P.ncls = L.ncls;
    for (int c = 0; c <= L.ncls; ++c) P.seg_pos[c] = L.seg_pos[c];
    for (int c = 0; c < L.ncls; ++c) P.seg_count[c] = L.seg_count[c];
    ET_TRY(ensure(ctx, ctx->rec, (size_t)L.npad * rec_floats(dim) * sizeof(float)));
    ET_TRY(ensure(ctx, ctx->prepkey, (size_t)L.npad * sizeof(uint32_t)));
    P.key_bits = std::min(20 / dim, 10);
    P.key = static_cast<uint32_t *>(ctx->prepkey.p);
    k_prep<TIn><<<grid, 256, 0, ctx->stream>>>(x, xbar, wx, wxbar, src, P, static_cast<float *>(ctx->rec.p));
    LAUNCH_CHECK();
    return ET_OK;
}

et_status run_prep(et_ctx *ctx, const void *x, const void *xbar, const double *wx, const double *wxbar, const int *src,
                   const Layout &L, int dim, et_dtype dtype, double sigma)
{
    if (dtype == ET_F32)
        return run_prep_t<float>(ctx, static_cast<const float *>(x), static_cast<const float *>(xbar), wx, wxbar, src, L, dim, sigma);
    return run_prep_t<double>(ctx, static_cast<const double *>(x), static_cast<const double *>(xbar), wx, wxbar, src, L, dim, sigma);
}

// ---- kernel dispatch over dim ----------------------------------------------------------------------------
#define DISPATCH_DIM(dim, ...)                                                   \
    switch (dim) {                                                               \
        case 1: { constexpr int D = 1; __VA_ARGS__; } break;                            \
        case 2: { constexpr int D = 2; __VA_ARGS__; } break;                            \
        case 3: { constexpr int D = 3; __VA_ARGS__; } break;                            \
        case 4: { constexpr int D = 4; __VA_ARGS__; } break;                            \
        case 5: { constexpr int D = 5; __VA_ARGS__; } break;                            \
        case 6: { constexpr int D = 6; __VA_ARGS__; } break;                            \
        case 7: { constexpr int D = 7; __VA_ARGS__; } break;                            \
        default: { constexpr int D = 8; __VA_ARGS__; } break;                           \
    }

template <typename K>
int resident_blocks(et_ctx *ctx, K kernel)
{
    int per_sm = 1;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, kThreads, 0) != cudaSuccess || per_sm < 1) per_sm = 1;
    return per_sm * ctx->num_sms;
}

constexpr int kRT = 4;    // rows per thread in K-T (i-tile = 1024 rows = kPad)
constexpr int kRRow = 2;  // rows per thread in K-ROW (i-tile = 512 rows)

et_status shard_sum(et_ctx *ctx, void *dev, int count, bool is_f64);

// K-T: class-pair sums into ctx->sums (device, kSumSlots doubles).  rec / tilecls default to the call's own layout;
// skip_mask drops class pairs (k_pairs_T); `booked` = false keeps the pass out of the per-kernel-class statistics (the
// escalation books its own time).
// Distance arithmetic of k_pairs_T (et_kernels.cuh): the Gram form when it pays -- dim >= 4, where the difference form is
// bound by the FP32 pipe (2 dim + 1 > 8 lane-ops per pair against 16 MUFU per clock and SM; measured at dim = 2: 14.9 vs
// 14.5 pairs/clk/SM, at dim = 5: 9.1 vs 11.4) -- and when the sample is large enough for its rounding noise to average far
// below the tolerance of T (>= kGramMinN events: the noise of T falls like 1 / N) and compact enough in units of sigma
// (|u|^2 <= kGramMaxU2: a per-pair error of psi below 4e-6); else differences.  ET_OPT_DISTANCE overrides.
constexpr long long kGramMinN = 4096;
constexpr double kGramMaxU2 = 48.0;
bool use_gram(const et_ctx *ctx, const Layout &L, int dim)
{
    if (ctx->opt_distance == 1) return false;
    if (ctx->opt_distance == 2) return ctx->umax2 <= 96.0;  // beyond, 2^(|u_i|^2) times a 128-term sum leaves the fp32 range
    return dim >= 4 && L.N >= kGramMinN && ctx->umax2 <= kGramMaxU2;
}

et_status run_pairs_T(et_ctx *ctx, const Layout &L, int dim, const float *rec = nullptr, const uint8_t *tilecls = nullptr,
                      unsigned skip_mask = 0u, bool booked = true)
{
    if (!rec) rec = static_cast<const float *>(ctx->rec.p);
    if (!tilecls) tilecls = static_cast<const uint8_t *>(ctx->tilecls.p);
    const int nT = (int)(L.npad / (kThreads * kRT));
    const long long nunits = (long long)nT * (nT + 1) / 2;
    ET_TRY(ensure(ctx, ctx->sums, kSumSlots * sizeof(double)));
    if (booked) ET_TRY(span_begin(ctx, 2));
    const bool gram = use_gram(ctx, L, dim);
    ctx->stats.distance_form = gram ? 2 : 1;
    DISPATCH_DIM(dim, {
        int grid = gram ? resident_blocks(ctx, k_pairs_T<D, kRT, true>) : resident_blocks(ctx, k_pairs_T<D, kRT, false>);
        const long long mine = (nunits - ctx->shard_rank + ctx->shard_world - 1) / ctx->shard_world;  // units of this rank
        if ((long long)grid > mine) grid = (int)std::max<long long>(mine, 1);
        ET_TRY(ensure(ctx, ctx->partials, (size_t)grid * kSumSlots * sizeof(double)));
        if (gram)
            k_pairs_T<D, kRT, true><<<grid, kThreads, 0, ctx->stream>>>(rec, nT, tilecls, nunits, skip_mask, ctx->shard_rank, ctx->shard_world,
                                                                       static_cast<double *>(ctx->partials.p));
        else
            k_pairs_T<D, kRT, false><<<grid, kThreads, 0, ctx->stream>>>(rec, nT, tilecls, nunits, skip_mask, ctx->shard_rank, ctx->shard_world,
                                                                        static_cast<double *>(ctx->partials.p));
        LAUNCH_CHECK();
        k_reduce_cols<<<1, 32, 0, ctx->stream>>>(static_cast<const double *>(ctx->partials.p), grid, kSumSlots,
                                                 static_cast<double *>(ctx->sums.p));
        LAUNCH_CHECK();
    });
    if (booked) ET_TRY(span_end(ctx, 2, &ctx->acc_pairs_ms, KC_T, 1, L.N * (L.N - 1) / 2 * (2 * dim + 1)));
    ctx->stats.pair_evals += nunits * (long long)(kThreads * kRT) * (kThreads * kRT) / ctx->shard_world;
    if (ctx->shard_world > 1) ET_TRY(shard_sum(ctx, ctx->sums.p, kSumSlots, true));
    return ET_OK;
}

// K-T for nsig sigmas in one pass (records scaled for sigmas[0]): class-pair sums into ctx->sums[s * kSumSlots + slot].
template <int NS>
et_status run_pairs_T_multi_ns(et_ctx *ctx, const Layout &L, int dim, const float *rho_dev)
{
    const int nT = (int)(L.npad / (kThreads * kRT));
    const long long nunits = (long long)nT * (nT + 1) / 2;
    DISPATCH_DIM(dim, {
        int grid = resident_blocks(ctx, k_pairs_T_multi<D, kRT, NS>);
        if ((long long)grid > nunits) grid = (int)nunits;
        ET_TRY(ensure(ctx, ctx->partials, (size_t)grid * NS * kSumSlots * sizeof(double)));
        k_pairs_T_multi<D, kRT, NS><<<grid, kThreads, 0, ctx->stream>>>(static_cast<const float *>(ctx->rec.p), nT,
                                                                       static_cast<const uint8_t *>(ctx->tilecls.p), nunits, rho_dev,
                                                                       static_cast<double *>(ctx->partials.p));
        LAUNCH_CHECK();
        k_reduce_cols<<<(NS * kSumSlots + 31) / 32, 32, 0, ctx->stream>>>(static_cast<const double *>(ctx->partials.p), grid, NS * kSumSlots,
                                                                         static_cast<double *>(ctx->sums.p));
        LAUNCH_CHECK();
    });
    ctx->stats.pair_evals += nunits * (long long)(kThreads * kRT) * (kThreads * kRT);
    return ET_OK;
}

// K-ROW: rowsum[c][row] for all rows.
// Grid of the CUDA-core permutation sums (grid_term, kFlushJ): step G = 2^(e + k - 24) with 2^e >= max |w| and
// 2^k >= min(N, kFlushJ), the most terms of one fp32 partial sum that can be non-zero; magic = 1.5 * 2^23 G.
double perm32_grid(const et_ctx *ctx, long long N)
{
    const double wabs = std::max(std::fabs(ctx->wmax), std::fabs(ctx->wmin));
    int e = 0, k = 0;
    if (std::frexp(wabs > 0 ? wabs : 1.0, &e) == 0.5) --e;  // wabs = m 2^e, 0.5 <= m < 1: the smallest e with 2^e >= wabs
    while ((1ll << k) < std::min<long long>(N, kFlushJ)) ++k;
    return std::ldexp(1.0, e + k - 24);
}

template <int C>
et_status run_pairs_rows_c(et_ctx *ctx, const Layout &L, int dim, float magic)
{
    const int nT = (int)(L.npad / (kThreads * kRRow));
    RowSegs segs{};
    for (int c = 0; c <= C; ++c) segs.jt_begin[c] = (int)(L.seg_pos[c] / kTileJ);
    ET_TRY(ensure(ctx, ctx->rowsum, (size_t)C * L.npad * sizeof(double)));
    ET_TRY(ensure(ctx, ctx->counter, sizeof(int)));
    CUDA_TRY(cudaMemsetAsync(ctx->counter.p, 0, sizeof(int), ctx->stream));
    ET_TRY(span_begin(ctx, 2));
    DISPATCH_DIM(dim, {
        int grid = resident_blocks(ctx, k_pairs_rows<D, kRRow, C>);
        if (grid > nT) grid = nT;
        k_pairs_rows<D, kRRow, C><<<grid, kThreads, 0, ctx->stream>>>(static_cast<const float *>(ctx->rec.p), nT, L.npad,
                                                                    static_cast<const uint8_t *>(ctx->tilecls.p), segs, magic,
                                                                    static_cast<int *>(ctx->counter.p),
                                                                    static_cast<double *>(ctx->rowsum.p));
        LAUNCH_CHECK();
    });
    ET_TRY(span_end(ctx, 2, &ctx->acc_pairs_ms, KC_ROW, 1, L.N * (L.N - 1) / 2 * (2 * dim + 1)));
    ctx->stats.pair_evals += L.npad * L.npad;
    return ET_OK;
}
// on_grid: the permutation path (terms rounded to the grid); false: plain fp32 terms (et_row_sums)
et_status run_pairs_rows(et_ctx *ctx, const Layout &L, int dim, bool on_grid = true)
{
    const float magic = on_grid ? (float)(12582912.0 * perm32_grid(ctx, L.N)) : 0.0f;
    return L.ncls == 2 ? run_pairs_rows_c<2>(ctx, L, dim, magic) : run_pairs_rows_c<4>(ctx, L, dim, magic);
}

// ---- labels ----------------------------------------------------------------------------------------------
// Radix select of K*_p for every permutation into ctx->sel.
et_status run_label_select(et_ctx *ctx, long long N, long long n_x, int nperm, uint64_t seed)
{
    ET_TRY(ensure(ctx, ctx->sel, (size_t)nperm * sizeof(SelState)));
    ET_TRY(ensure(ctx, ctx->hist, (size_t)nperm * 256 * sizeof(unsigned int)));
    CUDA_TRY(cudaMemsetAsync(ctx->hist.p, 0, (size_t)nperm * 256 * sizeof(unsigned int), ctx->stream));
    k_sel_init<<<(nperm + 255) / 256, 256, 0, ctx->stream>>>(static_cast<SelState *>(ctx->sel.p), nperm, n_x);
    LAUNCH_CHECK();
    const int ev = 8;
    const long long p0 = ctx->opt_perm_offset;
    const unsigned ngroups = (unsigned)(((p0 + nperm - 1) >> 2) - (p0 >> 2) + 1);
    const dim3 grid((unsigned)((N + (long long)kThreads * ev - 1) / ((long long)kThreads * ev)), ngroups);
    auto hist_pass = [&](int pass) -> et_status {
        k_sel_hist<<<grid, kThreads, 0, ctx->stream>>>(N, nperm, p0, (uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32), pass,
                                                      static_cast<const SelState *>(ctx->sel.p),
                                                      static_cast<unsigned int *>(ctx->hist.p), ev);
        LAUNCH_CHECK();
        k_sel_pick<<<(nperm + 7) / 8, 256, 0, ctx->stream>>>(static_cast<SelState *>(ctx->sel.p),
                                                             static_cast<unsigned int *>(ctx->hist.p), nperm);
        LAUNCH_CHECK();
        return ET_OK;
    };
    for (int pass = 0; pass < 4; ++pass) ET_TRY(hist_pass(pass));   // the key32 half of the composites
    if (ctx->opt_label_select == 1) {
        for (int pass = 4; pass < 8; ++pass) ET_TRY(hist_pass(pass));
        return ET_OK;
    }
    // the index half: one sweep lists the events of the wanted key32 bucket (about one), k_sel_finish takes the rank-th index
    ET_TRY(ensure(ctx, ctx->selcand, (size_t)nperm * (kSelCand + 1) * sizeof(uint32_t) + 16));
    unsigned int *cand_cnt = static_cast<unsigned int *>(ctx->selcand.p);
    int *overflow = reinterpret_cast<int *>(cand_cnt + nperm);
    uint32_t *cand = reinterpret_cast<uint32_t *>(cand_cnt + nperm + 4);
    CUDA_TRY(cudaMemsetAsync(cand_cnt, 0, ((size_t)nperm + 4) * sizeof(uint32_t), ctx->stream));
    ET_TRY(ensure(ctx, ctx->selsave, (size_t)nperm * sizeof(SelState)));
    CUDA_TRY(cudaMemcpyAsync(ctx->selsave.p, ctx->sel.p, (size_t)nperm * sizeof(SelState), cudaMemcpyDeviceToDevice, ctx->stream));
    k_sel_collect<<<grid, kThreads, 0, ctx->stream>>>(N, nperm, p0, (uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32),
                                                     static_cast<const SelState *>(ctx->sel.p), cand_cnt, cand, ev);
    LAUNCH_CHECK();
    k_sel_finish<<<(nperm + 255) / 256, 256, 0, ctx->stream>>>(static_cast<SelState *>(ctx->sel.p), cand_cnt, cand, nperm, overflow);
    LAUNCH_CHECK();
    int ovf = 0;
    ET_TRY(ensure_pinned(ctx, 4096));
    CUDA_TRY(cudaMemcpyAsync(ctx->pinned, overflow, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
    CUDA_TRY(cudaStreamSynchronize(ctx->stream));
    memcpy(&ovf, ctx->pinned, sizeof(int));
    if (ovf != 0) {  // a bucket beyond kSelCand events: the four sweeps over the index half, from the saved state
        CUDA_TRY(cudaMemcpyAsync(ctx->sel.p, ctx->selsave.p, (size_t)nperm * sizeof(SelState), cudaMemcpyDeviceToDevice, ctx->stream));
        for (int pass = 4; pass < 8; ++pass) ET_TRY(hist_pass(pass));
    }
    return ET_OK;
}

// Internal masks: column 0 = observed labelling (pooled index < n_a), column p + 1 = permutation p;
// word g of padded row r at mask[g * npad + r]; padding rows are zero.
et_status run_labels_internal(et_ctx *ctx, const Layout &L, int nperm, uint64_t seed, int *nwords_out)
{
    const int nwords = (nperm + 1 + 31) / 32;
    ET_TRY(span_begin(ctx, 4));
    ET_TRY(run_label_select(ctx, L.N, L.n_a, nperm, seed));
    ET_TRY(ensure(ctx, ctx->mask, (size_t)nwords * L.npad * sizeof(uint32_t)));
    CUDA_TRY(cudaMemsetAsync(ctx->mask.p, 0, (size_t)nwords * L.npad * sizeof(uint32_t), ctx->stream));
    LabelOut lo{};
    lo.stride_g = L.npad;
    lo.stride_i = 1;
    lo.nseg = L.ncls;
    for (int c = 0; c <= L.ncls; ++c) lo.seg_first[c] = L.seg_first[c];
    for (int c = 0; c < L.ncls; ++c) lo.seg_pos[c] = L.seg_pos[c];
    const dim3 grid((unsigned)((L.N + kThreads - 1) / kThreads), (unsigned)nwords);
    k_label_write<<<grid, kThreads, 0, ctx->stream>>>(L.N, L.n_a, nperm, ctx->opt_perm_offset, 1, nwords, (uint32_t)(seed & 0xffffffffu),
                                                     (uint32_t)(seed >> 32), static_cast<const SelState *>(ctx->sel.p), lo,
                                                     static_cast<uint32_t *>(ctx->mask.p));
    LAUNCH_CHECK();
    ET_TRY(span_end(ctx, 4, &ctx->acc_labels_ms));
    *nwords_out = nwords;
    return ET_OK;
}

// ---- statistic kernels (H6) -------------------------------------------------------------------------------
struct DevT {
    et_result r;
    int status;  // 0 ok, ET_ERR_DEGENERATE
};

__device__ void form_result(double S_xx, double S_bb, double S_xb, double W, double Wbar, long long npairs, DevT *out)
{
    et_result r;
    r.S_xx = S_xx; r.S_bb = S_bb; r.S_xb = S_xb; r.W = W; r.Wbar = Wbar; r.n_pairs = npairs;
    if (!(W > 1.0) || !(Wbar > 1.0)) {
        r.T = r.T_xx = r.T_bb = r.T_xb = nan("");
        out->r = r;
        out->status = ET_ERR_DEGENERATE;
        return;
    }
    r.T_xx = S_xx / (W * (W - 1.0));
    r.T_bb = S_bb / (Wbar * (Wbar - 1.0));
    r.T_xb = S_xb / (W * Wbar);
    r.T = r.T_xx + r.T_bb - r.T_xb;
    out->r = r;
    out->status = 0;
}

// Eq. 2 from class-pair sums S[c1*4+c2] (c1 <= c2) and class weights; sample A = classes with bit set in mask_a.
// One thread.  Used for X vs Xbar (2 classes) and for the P-even / P-odd regroupings of the four classes.
__global__ void k_stat_from_sums(const double *__restrict__ S, const double *__restrict__ clsw, int ncls, unsigned mask_a,
                                 long long npairs, DevT *out)
{
    if (threadIdx.x || blockIdx.x) return;
    double sxx = 0, sbb = 0, sxb = 0, W = 0, Wb = 0;
    for (int c1 = 0; c1 < ncls; ++c1) {
        const bool a1 = mask_a >> c1 & 1u;
        (a1 ? W : Wb) += clsw[c1];
        for (int c2 = c1; c2 < ncls; ++c2) {
            const bool a2 = mask_a >> c2 & 1u;
            const double s = S[c1 * 4 + c2];
            if (a1 && a2) sxx += s;
            else if (!a1 && !a2) sbb += s;
            else sxb += s;
        }
    }
    form_result(sxx, sbb, sxb, W, Wb, npairs, out);
}

// class weights: clsw[c] = sum of w over the rows of class c (fixed order: tiles in order, then threads)
__global__ void __launch_bounds__(kThreads) k_tile_weights(const float *__restrict__ rec, int F, int dim, double *__restrict__ out)
{
    __shared__ double s[kThreads / 32];
    const long long base = (long long)blockIdx.x * kPad;
    double a = 0.0;
    for (int k = threadIdx.x; k < kPad; k += kThreads) a += (double)rec[(base + k) * F + dim];
    a = warp_sum(a);
    if ((threadIdx.x & 31) == 0) s[threadIdx.x >> 5] = a;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int w = 0; w < kThreads / 32; ++w) t += s[w];
        out[blockIdx.x] = t;
    }
}
// out[c] (or out[c1*4+c2] when ncol > 1) = sum over the tiles of class c of in[tile*ncol + k]
__global__ void k_reduce_by_class(const double *__restrict__ in, const uint8_t *__restrict__ tile_cls, int ntiles, int ncol,
                                  double *__restrict__ out)
{
    const int c = threadIdx.x / ncol, k = threadIdx.x % ncol;
    if (c >= kMaxCls) return;
    double s = 0.0;
    for (int t = 0; t < ntiles; ++t)
        if (tile_cls[t] == c) s += in[(long long)t * ncol + k];
    if (ncol == 1) out[c] = s;
    else out[c * 4 + k] = s;
}
// rowsum-derived class-pair matrix M[c1*4+c2] = sum_{i in c1} w_i rowsum[c2][i] -> unordered-pair sums
// S[c1*4+c2] (c1 <= c2): diagonal halved, off-diagonal the mean of the two orientations.
__global__ void k_sym_class_sums(const double *__restrict__ M, int ncls, double *__restrict__ S)
{
    if (threadIdx.x || blockIdx.x) return;
    for (int a = 0; a < 16; ++a) S[a] = 0.0;
    for (int c1 = 0; c1 < ncls; ++c1)
        for (int c2 = c1; c2 < ncls; ++c2)
            S[c1 * 4 + c2] = c1 == c2 ? 0.5 * M[c1 * 4 + c1] : 0.5 * (M[c1 * 4 + c2] + M[c2 * 4 + c1]);
}

// Guard band of the decision T_p > T_obs (reading R5 of DESIGN.md): 8 sigma of the noise of T_p - T_obs under the error
// model of the arithmetic.  Every pair's Psi_ij = w_i w_j psi_ij carries an independent absolute error of standard
// deviation `pair_err` (fp32 path: 2^-22 wabs^2 -- ex2.approx is good to 2 ulp and psi <= 1; tensor-core path: that and
// the 15-bit rounding), so var(T) = pair_err^2 [ pairs_xx / (W(W-1))^2 + pairs_bb / (Wb(Wb-1))^2 + pairs_xb / (W Wb)^2 ]
// and the difference of two labellings that share the psi values has twice that.  1e-13 of the term scale covers the
// fp64 summation order.  The achieved errors are asserted against this band in tests/test_gpu_parity.py.
constexpr double kPairErrF32 = 2.384185791015625e-07;  // 2^-22
__device__ double guard_band(double pair_err, double nA, double nB, double Wo, double Wb, double scale)
{
    const double var = 0.5 * nA * (nA - 1.0) / ((Wo * (Wo - 1.0)) * (Wo * (Wo - 1.0))) + 0.5 * nB * (nB - 1.0) / ((Wb * (Wb - 1.0)) * (Wb * (Wb - 1.0))) +
                       nA * nB / ((Wo * Wb) * (Wo * Wb));
    return 1e-13 * scale + 8.0 * 1.4142135623730951 * pair_err * sqrt(var);
}

// Permutations inside the guard band, for the escalation (finite T_p only; NaN permutations cannot be decided).
constexpr int kMaxNear = 64;
struct DevNear {
    int n_finite;          // near permutations with a finite T_p (all of them, also beyond kMaxNear)
    int n_nan;             // degenerate weighted splits (T_p = NaN)
    int idx[kMaxNear];     // local permutation indices of the first kMaxNear (unordered)
    double guard;          // the band used
    double guard_f32;      // the band of the fp32-pair / fp64-sum arithmetic (what the escalation certifies)
};

// Permutation statistic (H6): columns c = 0 (observed) and c = p + 1.  From Q_c, R_c, W_c, S = RW_all / 2, Wtot:
//   S_xx = Q, S_bb = S - R + Q, S_xb = R - 2Q  (SURVEY 8(a) identity), Eq. 2 with W = W_c, Wbar = Wtot - W_c.
// Then count = #{T_p > T_obs}, n_near = #{|T_p - T_obs| <= guard, or T_p NaN}.
struct DevPerm {
    et_perm_result r;
    int status;
};
__global__ void __launch_bounds__(256) k_perm_stat(const double *__restrict__ Q, const double *__restrict__ RW, int nwords, int nperm,
                                                  long long npairs, double nA, double nB, double wabs, double qstep, double *__restrict__ T_perm, DevPerm *out)
{
    // RW layout: [g][which][kRWCols]
    __shared__ DevT obs;
    __shared__ unsigned long long s_cnt, s_near;
    const double S = 0.5 * RW[0 * 2 * kRWCols + 0 * kRWCols + 32];
    const double Wtot = RW[0 * 2 * kRWCols + 1 * kRWCols + 32];
    if (threadIdx.x == 0) {
        const double q = Q[0], r = RW[0], w = RW[kRWCols];
        form_result(q, S - r + q, r - 2.0 * q, w, Wtot - w, npairs, &obs);
        s_cnt = 0ull;
        s_near = 0ull;
    }
    __syncthreads();
    const double Tobs = obs.r.T;
    // every term w_j psi_ij sits on the grid of step qstep / |w_i| (grid_term): a rounding error of variance qstep^2 / 12
    const double e32 = kPairErrF32 * wabs * wabs;
    const double guard = guard_band(sqrt(e32 * e32 + qstep * qstep / 12.0), nA, nB, obs.r.W, obs.r.Wbar, fabs(obs.r.T_xx) + fabs(obs.r.T_bb) + fabs(obs.r.T_xb));
    unsigned long long cnt = 0, near = 0;
    for (int p = threadIdx.x; p < nperm; p += blockDim.x) {
        const int c = p + 1, g = c >> 5, b = c & 31;
        const double q = Q[g * 32 + b], r = RW[(g * 2 + 0) * kRWCols + b], w = RW[(g * 2 + 1) * kRWCols + b];
        DevT t;
        form_result(q, S - r + q, r - 2.0 * q, w, Wtot - w, npairs, &t);
        T_perm[p] = t.r.T;
        if (t.status != 0) { near += 1; continue; }
        if (t.r.T > Tobs) cnt += 1;
        if (fabs(t.r.T - Tobs) <= guard) near += 1;
    }
    atomicAdd(&s_cnt, cnt);
    atomicAdd(&s_near, near);
    __syncthreads();
    if (threadIdx.x == 0) {
        out->r.observed = obs.r;
        out->r.count_gt = (long long)s_cnt;
        out->r.n_near = (long long)s_near;
        out->r.nperm = nperm;
        out->r.p_value = (double)s_cnt / (double)nperm;
        out->status = obs.status;
    }
    (void)nwords;
}

// class weights into ctx->clsw (kMaxCls doubles)
// Eq. 3 from the ten class-pair sums of the layout (X, Bx, Xbar, Bxbar) = classes (0, 1, 2, 3).
// S[c1*4+c2] holds unordered pairs within a class (the printed sums over i != j are twice that) and all pairs across.
struct DevBkg {
    et_bkg_result r;
    int status;
};
__global__ void k_stat_eq3(const double *__restrict__ S, double n, double nbar, double bs, double bsb, double b, double bbar,
                           long long npairs, DevBkg *out, double *T_out)
{
    if (threadIdx.x || blockIdx.x) return;
    if (T_out) *T_out = nan("");
    et_bkg_result r;
    const int order[10] = {0, 1, 2, 3, 5, 6, 7, 10, 11, 15};
    for (int k = 0; k < 10; ++k) r.S[k] = S[order[k]];
    r.w = n - b;
    r.wbar = nbar - bbar;
    r.n_pairs = npairs;
    if (!(r.w > 1.0) || !(r.wbar > 1.0)) {
        r.T = r.T_xx = r.T_bb = r.T_xb = nan("");
        out->r = r;
        out->status = ET_ERR_DEGENERATE;
        return;
    }
    const double t1 = 2.0 * S[0] - 2.0 * b / bs * S[1] + b * (b + 1.0) / (bs * (bs - 1.0)) * 2.0 * S[5];
    const double t2 = 2.0 * S[10] - 2.0 * bbar / bsb * S[11] + bbar * (bbar + 1.0) / (bsb * (bsb - 1.0)) * 2.0 * S[15];
    const double t3 = S[2] - bbar / bsb * S[3] - b / bs * S[6] + b * bbar / (bs * bsb) * S[7];
    r.T_xx = t1 / (2.0 * r.w * (r.w - 1.0));
    r.T_bb = t2 / (2.0 * r.wbar * (r.wbar - 1.0));
    r.T_xb = t3 / (r.w * r.wbar);
    r.T = r.T_xx + r.T_bb - r.T_xb;
    out->r = r;
    out->status = 0;
    if (T_out) *T_out = r.T;
}
// src[row] for class segments that are consecutive runs of the pooled source index (class c = sources
// seg_first[c] .. seg_first[c] + seg_count[c] - 1), -1 on padding rows
__global__ void k_src_runs(PrepParams P, const long long *__restrict__ unused, int *__restrict__ src)
{
    for (long long row = blockIdx.x * (long long)blockDim.x + threadIdx.x; row < P.npad; row += (long long)gridDim.x * blockDim.x) {
        int v = -1;
        long long first = 0;
        for (int c = 0; c < P.ncls; ++c) {
            if (row >= P.seg_pos[c] && row - P.seg_pos[c] < P.seg_count[c]) v = (int)(first + row - P.seg_pos[c]);
            first += P.seg_count[c];
        }
        src[row] = v;
    }
}

et_status run_class_weights(et_ctx *ctx, const Layout &L, int dim, const float *rec = nullptr, const uint8_t *tilecls = nullptr)
{
    if (!rec) rec = static_cast<const float *>(ctx->rec.p);
    if (!tilecls) tilecls = static_cast<const uint8_t *>(ctx->tilecls.p);
    const int nt = (int)(L.npad / kPad);
    ET_TRY(ensure(ctx, ctx->clssum, (size_t)nt * 4 * sizeof(double)));
    ET_TRY(ensure(ctx, ctx->clsw, kMaxCls * sizeof(double)));
    k_tile_weights<<<nt, kThreads, 0, ctx->stream>>>(rec, rec_floats(dim), dim, static_cast<double *>(ctx->clssum.p));
    LAUNCH_CHECK();
    k_reduce_by_class<<<1, kMaxCls, 0, ctx->stream>>>(static_cast<const double *>(ctx->clssum.p), tilecls, nt, 1,
                                                     static_cast<double *>(ctx->clsw.p));
    LAUNCH_CHECK();
    return ET_OK;
}

long long pairs_two(long long a, long long b) { return a * (a - 1) / 2 + b * (b - 1) / 2 + a * b; }

// Fetch a DevT / DevPerm from the device.
template <typename T>
et_status fetch(et_ctx *ctx, const void *dev, T *host)
{
    ET_TRY(ensure_pinned(ctx, 4096));
    CUDA_TRY(cudaMemcpyAsync(ctx->pinned, dev, sizeof(T), cudaMemcpyDeviceToHost, ctx->stream));
    CUDA_TRY(cudaStreamSynchronize(ctx->stream));
    memcpy(host, ctx->pinned, sizeof(T));
    return ET_OK;
}

// ---- unit-range shard: completing partial sums over ranks --------------------------------------------------
// buf[r * count + k] (r < world) -> dev[k] = sum over r in rank order; T = long long (exact) or double (fixed order).
template <typename T>
__global__ void k_sum_slices(const T *__restrict__ buf, int world, int count, T *__restrict__ dev)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= count) return;
    T s = 0;
    for (int r = 0; r < world; ++r) s += buf[(long long)r * count + k];
    dev[k] = s;
}
// dev[count] holds this rank's partial sums (8-byte values); on return it holds the sums over all ranks, identical on
// every rank: the caller's all-gather (et_set_shard) fills a host buffer [world][count], summed on the device in rank order.
et_status shard_sum(et_ctx *ctx, void *dev, int count, bool is_f64)
{
    if (ctx->shard_world <= 1) return ET_OK;
    const size_t slice = (size_t)count * 8, total = slice * ctx->shard_world;
    ET_TRY(ensure_pinned(ctx, 4096 + total));
    char *h = static_cast<char *>(ctx->pinned) + 4096;  // the first 4 KB are the scratch of fetch() and prep
    memset(h, 0, total);
    CUDA_TRY(cudaMemcpyAsync(h + slice * ctx->shard_rank, dev, slice, cudaMemcpyDeviceToHost, ctx->stream));
    CUDA_TRY(cudaStreamSynchronize(ctx->stream));
    if (ctx->shard_fn(ctx->shard_user, h, (int64_t)slice) != 0) return fail(ctx, ET_ERR_INVALID, "the all-gather callback of et_set_shard failed");
    ET_TRY(ensure(ctx, ctx->shardbuf, total));
    CUDA_TRY(cudaMemcpyAsync(ctx->shardbuf.p, h, total, cudaMemcpyHostToDevice, ctx->stream));
    if (is_f64)
        k_sum_slices<double><<<(count + 255) / 256, 256, 0, ctx->stream>>>(static_cast<const double *>(ctx->shardbuf.p), ctx->shard_world, count, static_cast<double *>(dev));
    else
        k_sum_slices<long long><<<(count + 255) / 256, 256, 0, ctx->stream>>>(static_cast<const long long *>(ctx->shardbuf.p), ctx->shard_world, count, static_cast<long long *>(dev));
    LAUNCH_CHECK();
    CUDA_TRY(cudaStreamSynchronize(ctx->stream));  // the pinned buffer is reused by the next call
    return ET_OK;
}

// ---- the two-sample T from prepared records ---------------------------------------------------------------
et_status do_T(et_ctx *ctx, const void *x, const double *wx, int64_t n, const void *xbar, const double *wxbar, int64_t nbar,
               int dim, et_dtype dtype, et_memspace mem, double sigma, et_result *out)
{
    ET_TRY(begin_call(ctx));
    const void *dx = nullptr, *dxb = nullptr, *dwx = nullptr, *dwb = nullptr;
    ET_TRY(stage_in(ctx, x, (size_t)n * dim * elem_size(dtype), mem, ctx->in_x, &dx));
    ET_TRY(stage_in(ctx, xbar, (size_t)nbar * dim * elem_size(dtype), mem, ctx->in_xbar, &dxb));
    ET_TRY(stage_in(ctx, wx, (size_t)n * 8, mem, ctx->in_wx, &dwx));
    ET_TRY(stage_in(ctx, wxbar, (size_t)nbar * 8, mem, ctx->in_wxbar, &dwb));
    Layout L;
    layout_two(L, n, nbar);
    ET_TRY(upload_tile_classes(ctx, L));
    ET_TRY(run_prep(ctx, dx, dxb, static_cast<const double *>(dwx), static_cast<const double *>(dwb), nullptr, L, dim, dtype, sigma));
    ET_TRY(run_class_weights(ctx, L, dim));
    ET_TRY(run_pairs_T(ctx, L, dim));
    ET_TRY(ensure(ctx, ctx->result, sizeof(DevPerm) + sizeof(DevT) * 4));
    k_stat_from_sums<<<1, 32, 0, ctx->stream>>>(static_cast<const double *>(ctx->sums.p), static_cast<const double *>(ctx->clsw.p),
                                                2, 0x1u, pairs_two(n, nbar), static_cast<DevT *>(ctx->result.p));
    LAUNCH_CHECK();
    DevT r;
    ET_TRY(fetch(ctx, ctx->result.p, &r));
    ET_TRY(end_call(ctx));
    if (r.status != 0) return fail(ctx, ET_ERR_DEGENERATE, "weighted normalisation degenerate: W = %g, Wbar = %g (need > 1)", r.r.W, r.r.Wbar);
    *out = r.r;
    return ET_OK;
}

// ---- permutation sums from prepared records + masks -------------------------------------------------------
et_status run_perm_sums(et_ctx *ctx, const Layout &L, int dim, int nwords)
{
    // Q: CUDA-core kernel, one launch per mask word
    const int nT = (int)(L.npad / (kThreads * 2));
    const long long nunits = (long long)nT * (nT + 1) / 2;
    ET_TRY(ensure(ctx, ctx->Q, (size_t)nwords * 32 * sizeof(double)));
    ET_TRY(span_begin(ctx, 2));
    const float magic = (float)(12582912.0 * perm32_grid(ctx, L.N));
    DISPATCH_DIM(dim, {
        int grid = resident_blocks(ctx, k_perm32<D>);
        if ((long long)grid > nunits) grid = (int)nunits;
        ET_TRY(ensure(ctx, ctx->partQ, (size_t)grid * 32 * sizeof(double)));
        for (int g = 0; g < nwords; ++g) {
            k_perm32<D><<<grid, kThreads, 0, ctx->stream>>>(static_cast<const float *>(ctx->rec.p),
                                                           static_cast<const uint32_t *>(ctx->mask.p) + (long long)g * L.npad, nT,
                                                           nunits, magic, static_cast<double *>(ctx->partQ.p));
            LAUNCH_CHECK();
            k_reduce_cols<<<1, 32, 0, ctx->stream>>>(static_cast<const double *>(ctx->partQ.p), grid, 32,
                                                     static_cast<double *>(ctx->Q.p) + g * 32);
            LAUNCH_CHECK();
        }
    });
    ET_TRY(span_end(ctx, 2, &ctx->acc_pairs_ms, KC_PERM32, nwords, (long long)nwords * (L.N * (L.N - 1) / 2) * (2 * dim + 32)));
    ctx->stats.pair_evals += (long long)nwords * nunits * (kThreads * 2LL) * (kThreads * 2LL);

    // R, W per column
    const int nchunk = 64;
    ET_TRY(ensure(ctx, ctx->partRW, (size_t)nwords * nchunk * 2 * kRWCols * sizeof(double)));
    ET_TRY(ensure(ctx, ctx->RW, (size_t)nwords * 2 * kRWCols * sizeof(double)));
    const dim3 grid_rw((unsigned)nchunk, (unsigned)nwords);
    if (L.ncls == 2)
        k_perm_RW<2><<<grid_rw, kThreads, 0, ctx->stream>>>(static_cast<const float *>(ctx->rec.p), rec_floats(dim), dim,
                                                           static_cast<const uint32_t *>(ctx->mask.p),
                                                           static_cast<const double *>(ctx->rowsum.p), L.npad, nchunk,
                                                           static_cast<double *>(ctx->partRW.p));
    else
        k_perm_RW<4><<<grid_rw, kThreads, 0, ctx->stream>>>(static_cast<const float *>(ctx->rec.p), rec_floats(dim), dim,
                                                           static_cast<const uint32_t *>(ctx->mask.p),
                                                           static_cast<const double *>(ctx->rowsum.p), L.npad, nchunk,
                                                           static_cast<double *>(ctx->partRW.p));
    LAUNCH_CHECK();
    // partRW[g][chunk][2*kRWCols] -> RW[g][2*kRWCols]: per word a column reduction over the chunks
    for (int g = 0; g < nwords; ++g) {
        k_reduce_cols<<<1, 96, 0, ctx->stream>>>(static_cast<const double *>(ctx->partRW.p) + (long long)g * nchunk * 2 * kRWCols,
                                                 nchunk, 2 * kRWCols, static_cast<double *>(ctx->RW.p) + (long long)g * 2 * kRWCols);
        LAUNCH_CHECK();
    }
    return ET_OK;
}

et_status finish_perm(et_ctx *ctx, int nwords, int64_t nperm, long long npairs, double nA, double nB, double *T_perm, et_perm_result *out)
{
    const double wabs_ = std::max(std::fabs(ctx->wmax), std::fabs(ctx->wmin));
    ET_TRY(ensure(ctx, ctx->tperm, (size_t)nperm * sizeof(double)));
    ET_TRY(ensure(ctx, ctx->result, sizeof(DevPerm) + sizeof(DevT) * 4));
    k_perm_stat<<<1, 256, 0, ctx->stream>>>(static_cast<const double *>(ctx->Q.p), static_cast<const double *>(ctx->RW.p), nwords,
                                            (int)nperm, npairs, nA, nB, wabs_, perm32_grid(ctx, (long long)(nA + nB)) * wabs_,
                                            static_cast<double *>(ctx->tperm.p), static_cast<DevPerm *>(ctx->result.p));
    LAUNCH_CHECK();
    DevPerm r;
    ET_TRY(fetch(ctx, ctx->result.p, &r));
    if (r.status != 0) return fail(ctx, ET_ERR_DEGENERATE, "weighted normalisation degenerate: W = %g, Wbar = %g (need > 1)", r.r.observed.W, r.r.observed.Wbar);
    CUDA_TRY(cudaMemcpyAsync(T_perm, ctx->tperm.p, (size_t)nperm * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    CUDA_TRY(cudaStreamSynchronize(ctx->stream));
    *out = r.r;
    return ET_OK;
}


// ---- tensor-core permutation sums (K-PERM-TC) -------------------------------------------------------------
// W_c of the TC layout for unit weights (chunk ch, column c at ch * 512 + c): see run_perm_tc_g
__global__ void k_fill_W_tc(int nchunks, int nperm, double nA, double n_second, double Ntot, double *__restrict__ W)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= nchunks * tc::kCols) return;
    const int ch = k / tc::kCols, c = k % tc::kCols;
    double w;
    if (c == 0) w = nA;
    else if (c == 1) w = n_second;
    else if (c == 2) w = Ntot;
    else w = ch * tc::kPermsPerChunk + c - tc::kSpecial < nperm ? nA : 0.0;
    W[k] = w;
}
// T for every label column of the TC layout (et_tc.cuh): chunk ch, column c at index ch * 512 + c.
__global__ void __launch_bounds__(256) k_perm_stat_tc(const double *__restrict__ Q, const double *__restrict__ R, const double *__restrict__ W,
                                                     int nperm, long long npairs_obs, long long npairs_second, double qstep, double egram, double wabs,
                                                     double nA, double nB, double *__restrict__ T_perm, DevPerm *out, DevT *second, DevNear *nearout)
{
    __shared__ DevT obs;
    __shared__ unsigned long long s_cnt, s_near;
    __shared__ int s_nfin, s_nnan;
    const double S = Q[2], Wtot = W[2];  // the all-ones column
    if (threadIdx.x == 0) {
        form_result(Q[0], S - R[0] + Q[0], R[0] - 2.0 * Q[0], W[0], Wtot - W[0], npairs_obs, &obs);
        DevT sec;
        form_result(Q[1], S - R[1] + Q[1], R[1] - 2.0 * Q[1], W[1], Wtot - W[1], npairs_second, &sec);
        *second = sec;
        s_cnt = 0ull;
        s_near = 0ull;
        s_nfin = 0;
        s_nnan = 0;
    }
    __syncthreads();
    const double Tobs = obs.r.T;
    // guard band (reading R5, guard_band above): on top of the fp32 error of psi every pair carries the rounding of
    // w_j psi_ij to the 15-bit grid of step qstep / |w_i|, an independent error of variance kQuantVar qstep^2
    const double scale = fabs(obs.r.T_xx) + fabs(obs.r.T_bb) + fabs(obs.r.T_xb);
    const double e32 = kPairErrF32 * wabs * wabs;
    const double guard = guard_band(sqrt(tc::kQuantVar * qstep * qstep + e32 * e32), nA, nB, obs.r.W, obs.r.Wbar, scale);
    // the band of the escalation's arithmetic (k_pairs_T): fp32 psi, plus the rounding noise of the Gram form when it is used
    if (threadIdx.x == 0) { nearout->guard = guard; nearout->guard_f32 = guard_band(sqrt(e32 * e32 + egram * egram), nA, nB, obs.r.W, obs.r.Wbar, scale); }
    unsigned long long cnt = 0, near = 0;
    for (int p = threadIdx.x; p < nperm; p += blockDim.x) {
        const int k = (p / tc::kPermsPerChunk) * tc::kCols + tc::kSpecial + p % tc::kPermsPerChunk;
        // S of the chunk the column lives in: identical integers in every chunk (same quantised Psi), use chunk 0
        const double q = Q[k], r = R[k], w = W[k];
        DevT t;
        form_result(q, S - r + q, r - 2.0 * q, w, Wtot - w, npairs_obs, &t);
        T_perm[p] = t.r.T;
        if (t.status != 0) { near += 1; atomicAdd(&s_nnan, 1); continue; }
        if (t.r.T > Tobs) cnt += 1;
        if (fabs(t.r.T - Tobs) <= guard) {
            near += 1;
            const int k = atomicAdd(&s_nfin, 1);
            if (k < kMaxNear) nearout->idx[k] = p;
        }
    }
    atomicAdd(&s_cnt, cnt);
    atomicAdd(&s_near, near);
    __syncthreads();
    if (threadIdx.x == 0) {
        out->r.observed = obs.r;
        out->r.count_gt = (long long)s_cnt;
        out->r.n_near = (long long)s_near;
        out->r.nperm = nperm;
        out->r.p_value = (double)s_cnt / (double)nperm;
        out->status = obs.status;
        nearout->n_finite = s_nfin;
        nearout->n_nan = s_nnan;
    }
}

// Escalation, statistic of one re-evaluated permutation: D = T_p - T_obs in the fp32-pair / fp64-sum arithmetic from the
// class-pair sums S[c1 * 4 + c2] of the four classes (a_obs, a_perm) = A (1,1), B (1,0), C (0,1), D (0,0) (k_esc_class):
//   T_obs = c_xx (AA + AB + BB) + c_bb (CC + CD + DD) - c_xb (AC + AD + BC + BD),   X = A + B observed,
//   T_p   = c_xx (AA + AC + CC) + c_bb (BB + BD + DD) - c_xb (AB + AD + BC + CD),   X = A + C permuted.
// Unweighted, the sample sizes and hence c_xx = 1/(n(n-1)), c_bb, c_xb are those of both labellings, AA, DD, AD, BC cancel
// and were not evaluated (skip mask): D = (c_xx + c_xb)(AC - AB) + (c_bb + c_xb)(BD - CD) + (c_xx - c_bb)(CC - BB).
// Weighted, W_p differs from W_obs: both T from all ten sums and the class weights.
constexpr unsigned kEscSkipMask = (1u << 0) | (1u << 3) | (1u << 6) | (1u << 15);  // AA, AD, BC, DD
__global__ void k_esc_stat(const double *__restrict__ S, const double *__restrict__ clsw, int weighted, double nA, double nB, double *out)
{
    if (threadIdx.x || blockIdx.x) return;
    if (!weighted) {
        const double cxx = 1.0 / (nA * (nA - 1.0)), cbb = 1.0 / (nB * (nB - 1.0)), cxb = 1.0 / (nA * nB);
        *out = (cxx + cxb) * (S[2] - S[1]) + (cbb + cxb) * (S[7] - S[11]) + (cxx - cbb) * (S[10] - S[5]);
        return;
    }
    DevT o, p;
    form_result(S[0] + S[1] + S[5], S[10] + S[11] + S[15], S[2] + S[3] + S[6] + S[7], clsw[0] + clsw[1], clsw[2] + clsw[3], 0, &o);
    form_result(S[0] + S[2] + S[10], S[5] + S[7] + S[15], S[1] + S[3] + S[6] + S[11], clsw[0] + clsw[2], clsw[1] + clsw[3], 0, &p);
    *out = (o.status == 0 && p.status == 0) ? p.r.T - o.r.T : nan("");
}
// Applies the escalated differences: T_perm[p] = T_obs + D_p (the reported T_obs stays that of the tensor-core pass, so
// that count_gt = #{T_perm > T_obs} holds for what the caller sees), recounts, n_near = undecidable permutations.
__global__ void __launch_bounds__(256) k_esc_apply(const DevNear *__restrict__ nr, const double *__restrict__ D, int nesc, int nperm,
                                                  double *__restrict__ T_perm, DevPerm *out)
{
    __shared__ unsigned long long s_cnt;
    __shared__ int s_near;
    const double Tobs = out->r.observed.T;
    if (threadIdx.x == 0) { s_cnt = 0ull; s_near = nr->n_nan + (nr->n_finite - nesc); }
    __syncthreads();
    if ((int)threadIdx.x < nesc) {
        const double d = D[threadIdx.x];
        double t = Tobs + d;
        if (d > 0.0 && !(t > Tobs)) t = nextafter(Tobs, Tobs + 1.0);
        if (d < 0.0 && !(t < Tobs)) t = nextafter(Tobs, Tobs - 1.0);
        T_perm[nr->idx[threadIdx.x]] = t;
        if (!(fabs(d) > nr->guard_f32)) atomicAdd(&s_near, 1);
    }
    __syncthreads();
    unsigned long long cnt = 0;
    for (int p = threadIdx.x; p < nperm; p += blockDim.x)
        if (T_perm[p] > Tobs) cnt += 1;
    atomicAdd(&s_cnt, cnt);
    __syncthreads();
    if (threadIdx.x == 0) {
        out->r.count_gt = (long long)s_cnt;
        out->r.n_near = s_near;
        out->r.p_value = (double)s_cnt / (double)nperm;
    }
}

template <int D, class G>
et_status launch_perm_tc(et_ctx *ctx, const tc::TCParams &P, int grid, bool weighted, bool skip)
{
    if (skip && weighted) {  // far K blocks are not evaluated (et_tc.cuh, SKIP)
        CUDA_TRY(cudaFuncSetAttribute(tc::k_perm_tc<D, true, G, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, G::smem_tc(D)));
        tc::k_perm_tc<D, true, G, true><<<grid, G::kThreadsTC, G::smem_tc(D), ctx->stream>>>(P);
    } else if (skip) {
        CUDA_TRY(cudaFuncSetAttribute(tc::k_perm_tc<D, false, G, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, G::smem_tc(D)));
        tc::k_perm_tc<D, false, G, true><<<grid, G::kThreadsTC, G::smem_tc(D), ctx->stream>>>(P);
    } else if (weighted) {
        CUDA_TRY(cudaFuncSetAttribute(tc::k_perm_tc<D, true, G>, cudaFuncAttributeMaxDynamicSharedMemorySize, G::smem_tc(D)));
        tc::k_perm_tc<D, true, G><<<grid, G::kThreadsTC, G::smem_tc(D), ctx->stream>>>(P);
    } else {
        CUDA_TRY(cudaFuncSetAttribute(tc::k_perm_tc<D, false, G>, cudaFuncAttributeMaxDynamicSharedMemorySize, G::smem_tc(D)));
        tc::k_perm_tc<D, false, G><<<grid, G::kThreadsTC, G::smem_tc(D), ctx->stream>>>(P);
    }
    LAUNCH_CHECK();
    return ET_OK;
}

// Guard-band escalation (SURVEY 7 hard part 3; PAPER.md:67 defines p as the fraction of permutation T values greater
// than the observed one): the permutations whose tensor-core T_p lies within the guard band of T_obs are re-evaluated in
// the fp32-pair / fp64-sum arithmetic of k_pairs_T, one pass each.  The records of the call's layout are regrouped into
// the four classes (a_obs, a_perm) of that permutation (k_esc_class, stable partition, k_esc_gather -- the psi values are
// those of et_T bit for bit), k_pairs_T evaluates the class-pair sums that do not cancel in T_p - T_obs (six of ten when
// unweighted: 5/8 of the pairs), k_esc_stat forms the difference and k_esc_apply recounts.  Needs ctx->sel (the select
// states of the labels), ctx->rec, ctx->tperm and the DevPerm / DevNear of k_perm_stat_tc.
et_status run_escalation(et_ctx *ctx, const Layout &L, int dim, int nperm, uint64_t seed, bool weighted)
{
    DevNear nr;
    ET_TRY(fetch(ctx, ctx->nearbuf.p, &nr));
    if (nr.n_finite == 0 || nr.n_finite > kMaxNear || nr.n_finite > ctx->opt_exact_p) return ET_OK;
    ET_TRY(span_begin(ctx, 6));
    const int F = rec_floats(dim);
    const long long N = L.N;
    const int nblk = (int)((N + kPartBlock - 1) / kPartBlock);
    ET_TRY(ensure(ctx, ctx->esccls, (size_t)N));
    ET_TRY(ensure(ctx, ctx->blkcnt, (size_t)nblk * 4 * sizeof(int)));
    ET_TRY(ensure(ctx, ctx->totals, 16 * sizeof(long long)));
    ET_TRY(ensure(ctx, ctx->escD, kMaxNear * sizeof(double)));
    LabelOut lo{};
    lo.nseg = L.ncls;
    for (int c = 0; c <= L.ncls; ++c) lo.seg_first[c] = L.seg_first[c];
    for (int c = 0; c < L.ncls; ++c) lo.seg_pos[c] = L.seg_pos[c];
    for (int k = 0; k < nr.n_finite; ++k) {
        const int p = nr.idx[k];
        k_esc_class<<<(unsigned)((N + kThreads - 1) / kThreads), kThreads, 0, ctx->stream>>>(
            N, L.n_a, ctx->opt_perm_offset + p, (uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32),
            static_cast<const SelState *>(ctx->sel.p) + p, static_cast<uint8_t *>(ctx->esccls.p));
        LAUNCH_CHECK();
        k_part_count<<<nblk, kPartBlock, 0, ctx->stream>>>(N, static_cast<const uint8_t *>(ctx->esccls.p), static_cast<int *>(ctx->blkcnt.p));
        LAUNCH_CHECK();
        k_part_scan<<<1, 32, 0, ctx->stream>>>(nblk, static_cast<int *>(ctx->blkcnt.p), static_cast<long long *>(ctx->totals.p));
        LAUNCH_CHECK();
        long long cnt[4];
        ET_TRY(fetch(ctx, ctx->totals.p, &cnt));
        Layout L4;
        layout_four(L4, L.n_a, N - L.n_a, cnt);
        ET_TRY(upload_tile_classes(ctx, L4, &ctx->tilecls2));
        ET_TRY(ensure(ctx, ctx->src, (size_t)L4.npad * sizeof(int)));
        ET_TRY(ensure(ctx, ctx->rec2, (size_t)L4.npad * F * sizeof(float)));
        k_fill_int<<<ctx->num_sms * 4, 256, 0, ctx->stream>>>(static_cast<int *>(ctx->src.p), L4.npad, -1);
        LAUNCH_CHECK();
        CUDA_TRY(cudaMemcpyAsync(static_cast<long long *>(ctx->totals.p) + 8, L4.seg_pos, 4 * sizeof(long long), cudaMemcpyHostToDevice, ctx->stream));
        CUDA_TRY(cudaStreamSynchronize(ctx->stream));  // L4 is a local
        k_part_scatter<<<nblk, kPartBlock, 0, ctx->stream>>>(N, static_cast<const uint8_t *>(ctx->esccls.p), static_cast<const int *>(ctx->blkcnt.p),
                                                            static_cast<const long long *>(ctx->totals.p) + 8, static_cast<int *>(ctx->src.p));
        LAUNCH_CHECK();
        k_esc_gather<<<ctx->num_sms * 4, 256, 0, ctx->stream>>>(static_cast<const float4 *>(ctx->rec.p), static_cast<const int *>(ctx->src.p), L4.npad,
                                                               F / 4, lo, static_cast<float4 *>(ctx->rec2.p));
        LAUNCH_CHECK();
        const float *rec2 = static_cast<const float *>(ctx->rec2.p);
        const uint8_t *tc2 = static_cast<const uint8_t *>(ctx->tilecls2.p);
        if (weighted) ET_TRY(run_class_weights(ctx, L4, dim, rec2, tc2));
        else ET_TRY(ensure(ctx, ctx->clsw, kMaxCls * sizeof(double)));
        ET_TRY(run_pairs_T(ctx, L4, dim, rec2, tc2, weighted ? 0u : kEscSkipMask, false));
        k_esc_stat<<<1, 32, 0, ctx->stream>>>(static_cast<const double *>(ctx->sums.p), static_cast<const double *>(ctx->clsw.p), weighted ? 1 : 0,
                                              (double)L.n_a, (double)(N - L.n_a), static_cast<double *>(ctx->escD.p) + k);
        LAUNCH_CHECK();
    }
    k_esc_apply<<<1, 256, 0, ctx->stream>>>(static_cast<const DevNear *>(ctx->nearbuf.p), static_cast<const double *>(ctx->escD.p), nr.n_finite, nperm,
                                            static_cast<double *>(ctx->tperm.p), static_cast<DevPerm *>(ctx->result.p));
    LAUNCH_CHECK();
    double ms = 0;
    ET_TRY(span_end(ctx, 6, &ms));
    ctx->stats.ms_escalation += ms;
    ctx->stats.n_escalated += nr.n_finite;
    return ET_OK;
}

// Labels (TC layout), the contraction for every 512-column chunk, W_c, then the statistic.
// lab2_classes: class segments that form sample X of the second labelling (column 1).  G: geometry of k_perm_tc (et_tc.cuh).
template <class G>
et_status run_perm_tc_g(et_ctx *ctx, const Layout &L, int dim, int nperm, uint64_t seed, bool weighted, unsigned lab2_classes,
                        long long npairs_obs, long long npairs_second, double *T_perm, et_perm_result *out, et_result *second,
                        bool reuse_labels)
{
    const int nchunks = (nperm + tc::kPermsPerChunk - 1) / tc::kPermsPerChunk;
    const int words_total = nchunks * tc::kWordsPerChunk;
    // labels (reuse_labels: ctx->sel and ctx->maskT still hold those of the same (layout, nperm, seed), written by the
    // previous sigma of et_permutation_test_sigmas)
    ET_TRY(span_begin(ctx, 4));
    // the j range of the contraction is padded to whole K blocks: rows npad .. npadK - 1 carry zero labels and zero records
    const long long npadK = (L.npad + G::kKB - 1) / G::kKB * G::kKB;
    LabelOut lo{};
    lo.nseg = L.ncls;
    for (int c = 0; c <= L.ncls; ++c) lo.seg_first[c] = L.seg_first[c];
    for (int c = 0; c < L.ncls; ++c) lo.seg_pos[c] = L.seg_pos[c];
    // row order of the contraction (et_tc.cuh): Morton order inside every class segment.  With reuse_labels the order that
    // the labels were written in is kept (the keys of another sigma could round differently).
    // Unit weights: every pair enters once with a symmetric quantised psi, so the integer sums do not depend on the row
    // order at all.  With weights Psi_ij = w_j psi_ij is rounded per ordered pair, so the order shows in the last bits of the
    // sums (far inside the guard band); the keys come from the input coordinates and do not depend on sigma, so a sigma
    // scan and its single calls still agree bit for bit.
    if (!reuse_labels) ctx->tc_sorted = ctx->opt_tc_order != 0;
    const float *recT = static_cast<const float *>(ctx->rec.p);
    if (ctx->tc_sorted) {
        const int F4 = rec_floats(dim) / 4;
        ET_TRY(ensure(ctx, ctx->tcorder, (size_t)L.npad * sizeof(int)));
        ET_TRY(ensure(ctx, ctx->tcinv, (size_t)L.npad * sizeof(int)));
        ET_TRY(ensure(ctx, ctx->recS, (size_t)L.npad * rec_floats(dim) * sizeof(float)));
        if (!reuse_labels) {
            ET_TRY(ensure(ctx, ctx->tckey, (size_t)L.npad * sizeof(uint32_t)));
            ET_TRY(ensure(ctx, ctx->tckey2, (size_t)L.npad * sizeof(uint32_t)));
            ET_TRY(ensure(ctx, ctx->tcidx, (size_t)L.npad * sizeof(int)));
            // keys (k_prep) into (tckey2, tcorder); pass 1 -> (tckey, tcidx); pass 2 -> (tckey2, tcorder): the order ends in tcorder
            tc::k_key_iota<<<(unsigned)((L.npad + kThreads - 1) / kThreads), kThreads, 0, ctx->stream>>>(
                static_cast<const uint32_t *>(ctx->prepkey.p), L.npad, static_cast<uint32_t *>(ctx->tckey2.p), static_cast<int *>(ctx->tcorder.p));
            LAUNCH_CHECK();
            // at most 4096 tiles (one warp each) of at least 4096 elements
            long long tile = std::max<long long>(4096, (L.npad + 4095) / 4096);
            tile = (tile + 31) / 32 * 32;
            const long long ntiles = (L.npad + tile - 1) / tile, nhist = (long long)tc::kRsBins * ntiles;
            ET_TRY(ensure(ctx, ctx->rshist, (size_t)nhist * sizeof(uint32_t)));
            uint32_t *ka = static_cast<uint32_t *>(ctx->tckey2.p), *kb2 = static_cast<uint32_t *>(ctx->tckey.p);
            int *va = static_cast<int *>(ctx->tcorder.p), *vb = static_cast<int *>(ctx->tcidx.p);
            const unsigned rs_grid = (unsigned)((ntiles + tc::kRsWarps - 1) / tc::kRsWarps);
            for (int pass = 0; pass < 2; ++pass) {
                tc::k_rs_hist<<<rs_grid, 32 * tc::kRsWarps, 0, ctx->stream>>>(ka, L.npad, pass * tc::kRsBits, tile, ntiles, static_cast<uint32_t *>(ctx->rshist.p));
                LAUNCH_CHECK();
                tc::k_rs_scan<<<1, 1024, 0, ctx->stream>>>(static_cast<uint32_t *>(ctx->rshist.p), nhist);
                LAUNCH_CHECK();
                tc::k_rs_scatter<<<rs_grid, 32 * tc::kRsWarps, 0, ctx->stream>>>(ka, va, L.npad, pass * tc::kRsBits, tile, ntiles,
                                                                             static_cast<const uint32_t *>(ctx->rshist.p), kb2, vb);
                LAUNCH_CHECK();
                std::swap(ka, kb2);
                std::swap(va, vb);
            }
        }
        tc::k_order_gather<<<ctx->num_sms * 8, 256, 0, ctx->stream>>>(static_cast<const float4 *>(ctx->rec.p), static_cast<const int *>(ctx->tcorder.p), L.npad, F4,
                                                                    static_cast<int *>(ctx->tcinv.p), static_cast<float4 *>(ctx->recS.p));
        LAUNCH_CHECK();
        recT = static_cast<const float *>(ctx->recS.p);
    }
    if (!reuse_labels) {
        ET_TRY(run_label_select(ctx, L.N, L.n_a, nperm, seed));
        ET_TRY(ensure(ctx, ctx->maskT, (size_t)npadK * words_total * sizeof(uint32_t)));
        CUDA_TRY(cudaMemsetAsync(ctx->maskT.p, 0, (size_t)npadK * words_total * sizeof(uint32_t), ctx->stream));
        const dim3 grid((unsigned)((L.N + kThreads - 1) / kThreads), (unsigned)words_total);
        tc::k_label_write_tc<<<grid, kThreads, 0, ctx->stream>>>(L.N, L.n_a, nperm, ctx->opt_perm_offset, (uint32_t)(seed & 0xffffffffu),
                                                                (uint32_t)(seed >> 32), static_cast<const SelState *>(ctx->sel.p), lo,
                                                                lab2_classes, words_total, ctx->tc_sorted ? static_cast<const int *>(ctx->tcinv.p) : nullptr,
                                                                static_cast<uint32_t *>(ctx->maskT.p));
        LAUNCH_CHECK();
    }
    ET_TRY(span_end(ctx, 4, &ctx->acc_labels_ms));

    // unit table: 256-row tile I (one CTA pair) against K blocks [4 I, NK), cut at the GLOBAL boundaries m Lmax so that
    // units of the same chunk m read the same label rows; full-length units go first, chunk by chunk (the ~74 clusters
    // then stream one chunk of the label matrix together and it is served from L2: DRAM traffic per launch at config 4
    // fell from 640 GB to the order of the matrix itself, profiles/r01d), then the shorter ones, longest first.
    // unit u -> cluster u % nclusters
    const int nclusters_max = ctx->num_sms / 2;
    const int nT = (int)(L.npad / tc::kTM2), NK = (int)(npadK / G::kKB);
    auto first_kb = [](int I) { return (long long)I * tc::kTM2 / G::kKB; };  // K block that holds the tile's first row
    long long total_kb = 0;
    for (int I = 0; I < nT; ++I) total_kb += NK - first_kb(I);
    // Exact skipping of far K blocks (et_tc.cuh): with the rows in Morton order, mark for every row tile the K blocks whose
    // bounding box is within the distance at which a quantised Psi can be non-zero; the SKIP kernel walks the marked ones
    // only.  Taken when at least 5 % of the blocks are unmarked (BASELINE config 4: < 1 %, the plain kernel runs).
    bool use_skip = false;
    const int bm_words = (NK + 31) / 32;
    long long marked_kb = total_kb;
    // (the bitmap is nT x NK bits: 15 MB at 2e6 rows, O(N^2); beyond 256 MB -- about 8e6 rows -- every block is evaluated)
    if (ctx->tc_sorted && ctx->opt_tc_skip != 0 && (size_t)nT * (size_t)bm_words * sizeof(uint32_t) <= ((size_t)256 << 20)) {
        const int F = rec_floats(dim);
        ET_TRY(ensure(ctx, ctx->tcboxes, ((size_t)nT + (size_t)NK) * 2 * tc::kMaxDimTC * sizeof(float)));
        ET_TRY(ensure(ctx, ctx->tcbitmap, (size_t)nT * bm_words * sizeof(uint32_t) + 16));
        float *tlo = static_cast<float *>(ctx->tcboxes.p), *thi = tlo + (size_t)nT * tc::kMaxDimTC;
        float *klo = thi + (size_t)nT * tc::kMaxDimTC, *khi = klo + (size_t)NK * tc::kMaxDimTC;
        unsigned long long *marked = reinterpret_cast<unsigned long long *>(static_cast<uint32_t *>(ctx->tcbitmap.p) + (size_t)nT * bm_words + ((size_t)nT * bm_words & 1));
        tc::k_row_boxes<<<(unsigned)((nT + 7) / 8), kThreads, 0, ctx->stream>>>(recT, F, dim, L.npad, tc::kTM2, nT, tlo, thi);
        LAUNCH_CHECK();
        tc::k_row_boxes<<<(unsigned)((NK + 7) / 8), kThreads, 0, ctx->stream>>>(recT, F, dim, L.npad, G::kKB, NK, klo, khi);
        LAUNCH_CHECK();
        CUDA_TRY(cudaMemsetAsync(marked, 0, sizeof(unsigned long long), ctx->stream));
        tc::k_tile_bitmap<<<(unsigned)nT, kThreads, 0, ctx->stream>>>(tlo, thi, klo, khi, dim, NK, G::kKB, bm_words,
                                                                    static_cast<uint32_t *>(ctx->tcbitmap.p), marked);
        LAUNCH_CHECK();
        unsigned long long m = 0;
        ET_TRY(ensure_pinned(ctx, 4096));
        CUDA_TRY(cudaMemcpyAsync(ctx->pinned, marked, sizeof(m), cudaMemcpyDeviceToHost, ctx->stream));
        CUDA_TRY(cudaStreamSynchronize(ctx->stream));
        memcpy(&m, ctx->pinned, sizeof(m));
        if ((double)m < 0.95 * (double)total_kb) { use_skip = true; marked_kb = (long long)m; }
    }
    // about 24 units per cluster and rank (ranks of a unit-range shard take every world-th unit of the same table)
    const long long nshare = (long long)nclusters_max * 24 * ctx->shard_world;
    long long Lmax = (total_kb + nshare - 1) / nshare;
    if (Lmax < 8) Lmax = 8;
    if (Lmax > G::kMaxUnitKB) Lmax = G::kMaxUnitKB;
    std::vector<tc::Unit> full, tail;
    for (long long m = 0; m * Lmax < NK; ++m)
        for (int I = 0; I < nT && first_kb(I) < (m + 1) * Lmax; ++I) {
            tc::Unit u{I, (int)std::max<long long>(first_kb(I), m * Lmax), (int)std::min<long long>(NK, (m + 1) * Lmax), 0};
            if (u.kb_end <= u.kb_begin) continue;
            (u.kb_end - u.kb_begin == Lmax ? full : tail).push_back(u);
        }
    std::stable_sort(tail.begin(), tail.end(), [](const tc::Unit &a, const tc::Unit &b) { return a.kb_end - a.kb_begin > b.kb_end - b.kb_begin; });
    full.insert(full.end(), tail.begin(), tail.end());
    if (ctx->shard_world > 1) {  // this rank's share: every world-th unit, so that all ranks stream the same label chunks
        std::vector<tc::Unit> mine;
        for (size_t k = (size_t)ctx->shard_rank; k < full.size(); k += (size_t)ctx->shard_world) mine.push_back(full[k]);
        full.swap(mine);
        total_kb = 0;
        for (const tc::Unit &u : full) total_kb += u.kb_end - u.kb_begin;
        if (full.empty()) full.push_back(tc::Unit{0, 0, 0, 0});  // an empty unit: the kernel's epilogue still writes zero partials
    }
    const int nunits = (int)full.size();
    ET_TRY(ensure(ctx, ctx->units, full.size() * sizeof(tc::Unit)));
    CUDA_TRY(cudaMemcpyAsync(ctx->units.p, full.data(), full.size() * sizeof(tc::Unit), cudaMemcpyHostToDevice, ctx->stream));
    CUDA_TRY(cudaStreamSynchronize(ctx->stream));  // `full` goes out of scope

    // quantisation scale: v ~ sc Psi, 0 <= v < 2^15 (unsigned hi digit) or |v| < 2^14 (signed hi digit)
    double sc;
    bool hi_signed = false;
    if (!weighted) sc = tc::kScaleUnsigned;
    else if (ctx->wmin >= 0.0) sc = tc::kScaleUnsigned / std::max(ctx->wmax, 1e-30);
    else { hi_signed = true; sc = tc::kScaleSigned / std::max(std::fabs(ctx->wmin), std::fabs(ctx->wmax)); }

    const int grid = 2 * std::min(nclusters_max, nunits);  // CTA pairs
    const size_t part_bytes = (size_t)grid * G::kProducerWarps * G::kEpiGroups * 32 * 2 * 8;
    ET_TRY(ensure(ctx, ctx->tcpart, part_bytes));
    ET_TRY(ensure(ctx, ctx->tcQ, (size_t)nchunks * tc::kCols * sizeof(double)));
    ET_TRY(ensure(ctx, ctx->tcR, (size_t)nchunks * tc::kCols * sizeof(double)));
    ET_TRY(ensure(ctx, ctx->tcraw, 2 * tc::kCols * 8));
    ET_TRY(span_begin(ctx, 2));
    const float scf = (float)(256.0 * sc);
    ET_TRY(ensure(ctx, ctx->recP, (size_t)(npadK / 2) * tc::pair_rec_f4(dim) * sizeof(float4)));
    CUDA_TRY(cudaMemsetAsync(ctx->recP.p, 0, (size_t)(npadK / 2) * tc::pair_rec_f4(dim) * sizeof(float4), ctx->stream));
    DISPATCH_DIM(dim, (tc::k_pair_records<D><<<(unsigned)((L.npad / 2 + kThreads - 1) / kThreads), kThreads, 0, ctx->stream>>>(
                          recT, L.npad / 2, scf, static_cast<float4 *>(ctx->recP.p))));
    LAUNCH_CHECK();
    long long cols_algo = 0, cols_exec = 0;
    for (int ch = 0; ch < nchunks; ++ch) {
        tc::TCParams P{};
        P.rec = recT;
        P.maskT = static_cast<const uint32_t *>(ctx->maskT.p);
        P.words_total = words_total;
        P.word0 = ch * tc::kWordsPerChunk;
        P.units = static_cast<const tc::Unit *>(ctx->units.p);
        P.nunits = nunits;
        P.sc256 = scf;
        P.magic = hi_signed ? tc::kMagicSigned : tc::kMagicUnsigned;
        P.hixor = hi_signed ? 0x80808080u : 0u;
        P.recP = static_cast<const float4 *>(ctx->recP.p);
        P.idesc_hi = tc::umma_idesc_i8(hi_signed);
        // label columns of this launch: the three special ones and up to 509 permutations; 256 or fewer need one accumulator
        const int cols_used = tc::kSpecial + std::min(tc::kPermsPerChunk, nperm - ch * tc::kPermsPerChunk);
        P.nq = cols_used <= 256 ? 1 : 2;
        cols_algo += ch == 0 ? cols_used : cols_used - tc::kSpecial;  // the special columns are algorithmic work once
        cols_exec += 256 * P.nq;
        P.partial = ctx->tcpart.p;
        P.bitmap = use_skip ? static_cast<const uint32_t *>(ctx->tcbitmap.p) : nullptr;
        P.bm_words = bm_words;
        DISPATCH_DIM(dim, ET_TRY((launch_perm_tc<D, G>(ctx, P, grid, weighted, use_skip))));
        // the scale actually applied is the fp32 value of 256 sc
        const double inv_sc = 256.0 / (double)P.sc256;
        if (weighted) tc::k_tc_reduce<true, G><<<2, 256, 0, ctx->stream>>>(ctx->tcpart.p, grid, ctx->tcraw.p);
        else tc::k_tc_reduce<false, G><<<2, 256, 0, ctx->stream>>>(ctx->tcpart.p, grid, ctx->tcraw.p);
        LAUNCH_CHECK();
        ET_TRY(shard_sum(ctx, ctx->tcraw.p, 2 * tc::kCols, weighted));  // exact int64 (or fp64) column sums over the ranks
        if (weighted)
            tc::k_tc_scale<true><<<2, 256, 0, ctx->stream>>>(ctx->tcraw.p, inv_sc, static_cast<double *>(ctx->tcQ.p) + ch * tc::kCols,
                                                           static_cast<double *>(ctx->tcR.p) + ch * tc::kCols);
        else
            tc::k_tc_scale<false><<<2, 256, 0, ctx->stream>>>(ctx->tcraw.p, inv_sc, static_cast<double *>(ctx->tcQ.p) + ch * tc::kCols,
                                                            static_cast<double *>(ctx->tcR.p) + ch * tc::kCols);
        LAUNCH_CHECK();
    }
    {
        const long long pairs = L.N * (L.N - 1) / 2;
        // algorithmic work (et.h): 2 digits x 2 ops per (pair, label column) over the columns the test needs -- the
        // permutations plus observed / second labelling / ones once; the executed count (padded accumulators, the
        // special columns repeated in every chunk) is kept beside it
        // with far K blocks skipped the work is that of the evaluated blocks (the rest is known to be exactly zero)
        const double evaluated = use_skip ? (double)marked_kb / (double)total_kb : 1.0;
        ET_TRY(span_end(ctx, 2, &ctx->acc_pairs_ms, KC_PERMTC, nchunks, (int64_t)(2.0 * 2 * (double)pairs * (double)cols_algo * evaluated)));
        ctx->stats.dominant_ops_executed = (int64_t)(2.0 * 2 * (double)pairs * (double)cols_exec * evaluated);
        ctx->stats.pair_evals += (long long)nchunks * (use_skip && ctx->shard_world == 1 ? marked_kb : total_kb) * tc::kTM2 * G::kKB;
    }

    // W_c
    const int nchunkW = 64;
    ET_TRY(ensure(ctx, ctx->tcWpart, (size_t)words_total * nchunkW * 32 * sizeof(double)));
    ET_TRY(ensure(ctx, ctx->tcW, (size_t)words_total * 32 * sizeof(double)));
    if (!weighted) {
        // unit weights: W_c is the number of ones of the column, known without a pass over the 256 MB of labels -- n_a for the
        // observed labelling and for every permutation (reading R4 preserves the sizes; pin P10), the size of the second
        // labelling's sample, N for the all-ones column: the same doubles k_perm_W_tc sums up
        long long n_second = 0;
        for (int c = 0; c < L.ncls; ++c)
            if (lab2_classes >> c & 1u) n_second += L.seg_count[c];
        k_fill_W_tc<<<(nchunks * tc::kCols + 255) / 256, 256, 0, ctx->stream>>>(nchunks, nperm, (double)L.n_a, (double)n_second, (double)L.N,
                                                                                 static_cast<double *>(ctx->tcW.p));
        LAUNCH_CHECK();
    } else {
        const dim3 gridW((unsigned)nchunkW, (unsigned)words_total);
        tc::k_perm_W_tc<<<gridW, kThreads, 0, ctx->stream>>>(recT, rec_floats(dim), dim,
                                                            static_cast<const uint32_t *>(ctx->maskT.p), words_total, L.npad, nchunkW,
                                                            static_cast<double *>(ctx->tcWpart.p));
        LAUNCH_CHECK();
        for (int wd = 0; wd < words_total; ++wd) {
            k_reduce_cols<<<1, 32, 0, ctx->stream>>>(static_cast<const double *>(ctx->tcWpart.p) + (long long)wd * nchunkW * 32, nchunkW, 32,
                                                     static_cast<double *>(ctx->tcW.p) + wd * 32);
            LAUNCH_CHECK();
        }
    }
    // statistic
    const double wabs = std::max(std::fabs(ctx->wmax), std::fabs(ctx->wmin));
    const double qstep = wabs / sc;  // one rounding step of w_j psi_ij, times |w_i| <= wabs
    const double egram = use_gram(ctx, L, dim) ? kGramErr * ctx->umax2 * wabs * wabs : 0.0;  // error of Psi_ij in the escalation's k_pairs_T
    ET_TRY(ensure(ctx, ctx->tperm, (size_t)nperm * sizeof(double)));
    ET_TRY(ensure(ctx, ctx->result, sizeof(DevPerm) + sizeof(DevT) * 4));
    DevT *dev_second = reinterpret_cast<DevT *>(static_cast<char *>(ctx->result.p) + sizeof(DevPerm));
    ET_TRY(ensure(ctx, ctx->nearbuf, sizeof(DevNear)));
    k_perm_stat_tc<<<1, 256, 0, ctx->stream>>>(static_cast<const double *>(ctx->tcQ.p), static_cast<const double *>(ctx->tcR.p),
                                               static_cast<const double *>(ctx->tcW.p), nperm, npairs_obs, npairs_second, qstep, egram, wabs,
                                               (double)L.n_a, (double)(L.N - L.n_a),
                                               static_cast<double *>(ctx->tperm.p), static_cast<DevPerm *>(ctx->result.p), dev_second,
                                               static_cast<DevNear *>(ctx->nearbuf.p));
    LAUNCH_CHECK();
    DevPerm r;
    ET_TRY(fetch(ctx, ctx->result.p, &r));
    if (r.status != 0) return fail(ctx, ET_ERR_DEGENERATE, "weighted normalisation degenerate: W = %g, Wbar = %g (need > 1)", r.r.observed.W, r.r.observed.Wbar);
    ctx->stats.n_near_before = r.r.n_near;
    if (r.r.n_near > 0 && ctx->opt_exact_p > 0) {
        ET_TRY(run_escalation(ctx, L, dim, nperm, seed, weighted));
        ET_TRY(fetch(ctx, ctx->result.p, &r));
    }
    DevT sec;
    ET_TRY(fetch(ctx, dev_second, &sec));
    CUDA_TRY(cudaMemcpyAsync(T_perm, ctx->tperm.p, (size_t)nperm * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    CUDA_TRY(cudaStreamSynchronize(ctx->stream));
    *out = r.r;
    if (second) *second = sec.r;
    return ET_OK;
}

// Geometry by dimension (et_tc.cuh): the 16-producer-warp / 128-j layout while the i rows fit its 96 registers.
et_status run_perm_tc(et_ctx *ctx, const Layout &L, int dim, int nperm, uint64_t seed, bool weighted, unsigned lab2_classes,
                      long long npairs_obs, long long npairs_second, double *T_perm, et_perm_result *out, et_result *second,
                      bool reuse_labels = false)
{
    if (dim <= 5)
        return run_perm_tc_g<tc::Geo128>(ctx, L, dim, nperm, seed, weighted, lab2_classes, npairs_obs, npairs_second, T_perm, out, second, reuse_labels);
    return run_perm_tc_g<tc::Geo96>(ctx, L, dim, nperm, seed, weighted, lab2_classes, npairs_obs, npairs_second, T_perm, out, second, reuse_labels);
}

bool use_tc(const et_ctx *ctx, const Layout &L)
{
    if (ctx->opt_perm_kernel == 1) return false;
    if (ctx->opt_perm_kernel == 2) return true;
    // >= 8192 padded rows: the 15-bit rounding noise of T (0.82 / 32766 / N) is then 8 sigma < 4e-8, inside the 1e-6
    // tolerance for every term scale >= 0.04, and the contraction beats the CUDA-core kernel (one pass per 32 columns) by
    // 5 - 10 x at 1000 permutations (measured at N = 2000 .. 16 000, profiles/r02_README.md)
    return L.npad >= 8192;
}

}  // namespace

// =============================================================================================== C ABI
extern "C" {

const char *et_version(void) { return "libet 0.1 (sm_100a)"; }

et_status et_create(et_ctx **out, int device, void *cuda_stream)
{
    if (!out) return ET_ERR_INVALID;
    *out = nullptr;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1 || device < 0 || device >= ndev) return ET_ERR_CUDA;
    et_ctx *ctx = new (std::nothrow) et_ctx();
    if (!ctx) return ET_ERR_NOMEM;
    ctx->device = device;
    bool ok = cudaSetDevice(device) == cudaSuccess;
    cudaDeviceProp prop;
    ok = ok && cudaGetDeviceProperties(&prop, device) == cudaSuccess;
    if (ok) ctx->num_sms = prop.multiProcessorCount;
    if (ok) {
        if (cuda_stream) { ctx->stream = static_cast<cudaStream_t>(cuda_stream); ctx->own_stream = false; }
        else { ok = cudaStreamCreateWithFlags(&ctx->stream, cudaStreamNonBlocking) == cudaSuccess; ctx->own_stream = ok; }
    }
    for (int i = 0; ok && i < 8; ++i) ok = cudaEventCreate(&ctx->ev[i]) == cudaSuccess;
    if (!ok) { et_destroy(ctx); return ET_ERR_CUDA; }
    *out = ctx;
    return ET_OK;
}

void et_destroy(et_ctx *ctx)
{
    if (!ctx) return;
    cudaSetDevice(ctx->device);
    if (ctx->stream) cudaStreamSynchronize(ctx->stream);
    Buf *bufs[] = {&ctx->in_x, &ctx->in_xbar, &ctx->in_wx, &ctx->in_wxbar, &ctx->in_mx, &ctx->in_mb, &ctx->in_aux, &ctx->rec,
                   &ctx->tilecls, &ctx->partials, &ctx->sums, &ctx->rowsum, &ctx->mask, &ctx->sel, &ctx->hist, &ctx->partQ,
                   &ctx->Q, &ctx->partRW, &ctx->RW, &ctx->mm, &ctx->flag, &ctx->counter, &ctx->src, &ctx->posx, &ctx->posb,
                   &ctx->blkcnt, &ctx->totals, &ctx->clsw, &ctx->clssum, &ctx->result, &ctx->tperm, &ctx->rows, &ctx->rowsout,
                   &ctx->count64, &ctx->maskT, &ctx->units, &ctx->tcpart, &ctx->tcQ, &ctx->tcR, &ctx->tcWpart, &ctx->tcW, &ctx->recP,
                   &ctx->shardbuf, &ctx->tcraw, &ctx->rec2, &ctx->tilecls2, &ctx->esccls, &ctx->escD, &ctx->nearbuf, &ctx->escw,
                   &ctx->scpcnt, &ctx->scpS, &ctx->selcand, &ctx->selsave, &ctx->tckey, &ctx->tckey2, &ctx->tcidx, &ctx->tcorder,
                   &ctx->tcinv, &ctx->recS, &ctx->rshist, &ctx->tcboxes, &ctx->tcbitmap, &ctx->prepkey};
    for (Buf *b : bufs)
        if (b->p) cudaFree(b->p);
    if (ctx->pinned) cudaFreeHost(ctx->pinned);
    for (int i = 0; i < 8; ++i)
        if (ctx->ev[i]) cudaEventDestroy(ctx->ev[i]);
    if (ctx->own_stream && ctx->stream) cudaStreamDestroy(ctx->stream);
    nvtx_close_all(ctx);
    delete ctx;
}

const char *et_last_error(const et_ctx *ctx) { return ctx ? ctx->err : "null context"; }

et_status et_set_option(et_ctx *ctx, et_option opt, int64_t value)
{
    if (!ctx) return ET_ERR_INVALID;
    if (opt == ET_OPT_PERM_KERNEL) {
        if (value < 0 || value > 2) return fail(ctx, ET_ERR_INVALID, "unknown permutation kernel %lld", (long long)value);
        ctx->opt_perm_kernel = value;
        return ET_OK;
    }
    if (opt == ET_OPT_PERM_OFFSET) {
        // the Philox counter word of reading R4 is (uint32)(p >> 2): permutation indices stay below 2^34
        if (value < 0 || value > (1ll << 34) - ET_MAX_NPERM) return fail(ctx, ET_ERR_INVALID, "permutation offset out of range (p0 + nperm must stay below 2^34)");
        ctx->opt_perm_offset = value;
        return ET_OK;
    }
    if (opt == ET_OPT_DISTANCE) {
        if (value < 0 || value > 2) return fail(ctx, ET_ERR_INVALID, "ET_OPT_DISTANCE must be 0, 1 or 2");
        ctx->opt_distance = value;
        return ET_OK;
    }
    if (opt == ET_OPT_TC_SKIP) {
        if (value < 0 || value > 1) return fail(ctx, ET_ERR_INVALID, "ET_OPT_TC_SKIP must be 0 or 1");
        ctx->opt_tc_skip = value;
        return ET_OK;
    }
    if (opt == ET_OPT_TC_ORDER) {
        if (value < 0 || value > 1) return fail(ctx, ET_ERR_INVALID, "ET_OPT_TC_ORDER must be 0 or 1");
        ctx->opt_tc_order = value;
        return ET_OK;
    }
    if (opt == ET_OPT_LABEL_SELECT) {
        if (value < 0 || value > 1) return fail(ctx, ET_ERR_INVALID, "ET_OPT_LABEL_SELECT must be 0 or 1");
        ctx->opt_label_select = value;
        return ET_OK;
    }
    if (opt == ET_OPT_EXACT_P) {
        if (value < 0 || value > kMaxNear) return fail(ctx, ET_ERR_INVALID, "ET_OPT_EXACT_P must be in 0..%d", kMaxNear);
        ctx->opt_exact_p = value;
        return ET_OK;
    }
    return fail(ctx, ET_ERR_INVALID, "unknown option %d", (int)opt);
}

et_status et_set_shard(et_ctx *ctx, int rank, int world, et_allgather_fn fn, void *user)
{
    if (!ctx) return ET_ERR_INVALID;
    if (world < 1 || world > 4096 || rank < 0 || rank >= world) return fail(ctx, ET_ERR_INVALID, "bad shard: rank %d of %d", rank, world);
    if (world > 1 && !fn) return fail(ctx, ET_ERR_INVALID, "a shard over %d ranks needs the all-gather callback", world);
    ctx->shard_rank = rank;
    ctx->shard_world = world;
    ctx->shard_fn = fn;
    ctx->shard_user = user;
    return ET_OK;
}

et_status et_get_stats(const et_ctx *ctx, et_stats *out)
{
    if (!ctx || !out) return ET_ERR_INVALID;
    *out = ctx->stats;
    return ET_OK;
}

et_status et_T(et_ctx *ctx, const void *x, int64_t n, const void *xbar, int64_t nbar, int dim, et_dtype dtype, et_memspace mem,
               double sigma, et_result *out)
{
    ET_TRY(check_common(ctx, x, n, xbar, nbar, dim, dtype, mem, sigma));
    if (!out) return fail(ctx, ET_ERR_INVALID, "null output");
    return do_T(ctx, x, nullptr, n, xbar, nullptr, nbar, dim, dtype, mem, sigma, out);
}

et_status et_T_weighted(et_ctx *ctx, const void *x, const double *wx, int64_t n, const void *xbar, const double *wxbar,
                        int64_t nbar, int dim, et_dtype dtype, et_memspace mem, double sigma, et_result *out)
{
    ET_TRY(check_common(ctx, x, n, xbar, nbar, dim, dtype, mem, sigma));
    if (!out || !wx || !wxbar) return fail(ctx, ET_ERR_INVALID, "null weights or output");
    return do_T(ctx, x, wx, n, xbar, wxbar, nbar, dim, dtype, mem, sigma, out);
}

et_status et_T_sigmas(et_ctx *ctx, const void *x, const double *wx, int64_t n, const void *xbar, const double *wxbar, int64_t nbar,
                      int dim, et_dtype dtype, et_memspace mem, const double *sigmas, int nsig, et_result *out)
{
    if (!ctx) return ET_ERR_INVALID;
    if (!sigmas || !out) return fail(ctx, ET_ERR_INVALID, "null sigmas or output");
    if (nsig < 1 || nsig > ET_MAX_SIGMAS) return fail(ctx, ET_ERR_INVALID, "nsig must be in 1..%d; got %d", ET_MAX_SIGMAS, nsig);
    for (int s = 0; s < nsig; ++s) ET_TRY(check_common(ctx, x, n, xbar, nbar, dim, dtype, mem, sigmas[s]));
    if ((wx == nullptr) != (wxbar == nullptr)) return fail(ctx, ET_ERR_INVALID, "weights: both NULL or both given");
    if (nsig == 1) return do_T(ctx, x, wx, n, xbar, wxbar, nbar, dim, dtype, mem, sigmas[0], out);
    // the exponent scale rho_s = (sigma_0 / sigma_s)^2 multiplies e (< 2^7 where psi matters): keep it within fp32 range
    for (int s = 1; s < nsig; ++s) {
        const double r = sigmas[0] / sigmas[s];
        if (!(r * r < 1e12) || !(r * r > 1e-12)) return fail(ctx, ET_ERR_SIGMA, "sigmas differ by more than a factor 1e6");
    }
    ET_TRY(begin_call(ctx));
    const void *dx = nullptr, *dxb = nullptr, *dwx = nullptr, *dwb = nullptr;
    ET_TRY(stage_in(ctx, x, (size_t)n * dim * elem_size(dtype), mem, ctx->in_x, &dx));
    ET_TRY(stage_in(ctx, xbar, (size_t)nbar * dim * elem_size(dtype), mem, ctx->in_xbar, &dxb));
    ET_TRY(stage_in(ctx, wx, (size_t)n * 8, mem, ctx->in_wx, &dwx));
    ET_TRY(stage_in(ctx, wxbar, (size_t)nbar * 8, mem, ctx->in_wxbar, &dwb));
    Layout L;
    layout_two(L, n, nbar);
    ET_TRY(upload_tile_classes(ctx, L));
    ET_TRY(run_prep(ctx, dx, dxb, static_cast<const double *>(dwx), static_cast<const double *>(dwb), nullptr, L, dim, dtype, sigmas[0]));
    ET_TRY(run_class_weights(ctx, L, dim));
    ET_TRY(ensure(ctx, ctx->sums, (size_t)ET_MAX_SIGMAS * kSumSlots * sizeof(double) + 64));
    float *rho_dev = reinterpret_cast<float *>(static_cast<double *>(ctx->sums.p) + ET_MAX_SIGMAS * kSumSlots);
    ET_TRY(ensure_pinned(ctx, 4096));
    float *rho_h = static_cast<float *>(ctx->pinned) + 512;
    for (int s = 0; s < nsig; ++s) rho_h[s] = (float)((sigmas[0] / sigmas[s]) * (sigmas[0] / sigmas[s]));
    CUDA_TRY(cudaMemcpyAsync(rho_dev, rho_h, nsig * sizeof(float), cudaMemcpyHostToDevice, ctx->stream));
    ET_TRY(span_begin(ctx, 2));
    if (nsig == 2) ET_TRY(run_pairs_T_multi_ns<2>(ctx, L, dim, rho_dev));
    else if (nsig == 3) ET_TRY(run_pairs_T_multi_ns<3>(ctx, L, dim, rho_dev));
    else ET_TRY(run_pairs_T_multi_ns<4>(ctx, L, dim, rho_dev));
    ET_TRY(span_end(ctx, 2, &ctx->acc_pairs_ms, KC_T, 1, L.N * (L.N - 1) / 2 * (2 * dim + 1 + 2 * (nsig - 1))));
    ET_TRY(ensure(ctx, ctx->result, sizeof(DevPerm) + sizeof(DevT) * 4 + sizeof(DevBkg)));
    for (int s = 0; s < nsig; ++s) {
        k_stat_from_sums<<<1, 32, 0, ctx->stream>>>(static_cast<const double *>(ctx->sums.p) + s * kSumSlots, static_cast<const double *>(ctx->clsw.p),
                                                    2, 0x1u, pairs_two(n, nbar), static_cast<DevT *>(ctx->result.p) + s);
        LAUNCH_CHECK();
    }
    DevT r[ET_MAX_SIGMAS];
    ET_TRY(ensure_pinned(ctx, 4096));
    CUDA_TRY(cudaMemcpyAsync(ctx->pinned, ctx->result.p, sizeof(DevT) * nsig, cudaMemcpyDeviceToHost, ctx->stream));
    CUDA_TRY(cudaStreamSynchronize(ctx->stream));
    memcpy(r, ctx->pinned, sizeof(DevT) * nsig);
    ET_TRY(end_call(ctx));
    for (int s = 0; s < nsig; ++s)
        if (r[s].status != 0) return fail(ctx, ET_ERR_DEGENERATE, "weighted normalisation degenerate: W = %g, Wbar = %g (need > 1)", r[s].r.W, r[s].r.Wbar);
    for (int s = 0; s < nsig; ++s) out[s] = r[s].r;
    return ET_OK;
}

}  // extern "C" (helpers of the Eq. 3 entry points follow)
namespace {

// Validation, staging, identity four-class layout (X, Bx, Xbar, Bxbar), records, one K-T pass and Eq. 3 of the observed
// samples.  Leaves the records in ctx->rec and the layout in L.
et_status bkg_observed(et_ctx *ctx, const void *x, int64_t n, const void *xbar, int64_t nbar, const void *bx, int64_t bs,
                       const void *bxbar, int64_t bsbar, double b, double bbar, int dim, et_dtype dtype, et_memspace mem, double sigma,
                       Layout &L, DevBkg &r)
{
    // the x side of the pooled source index is [x ; bx], the xbar side [xbar ; bxbar]
    const size_t row = (size_t)dim * elem_size(dtype);
    ET_TRY(ensure(ctx, ctx->in_x, (size_t)(n + bs) * row));
    ET_TRY(ensure(ctx, ctx->in_xbar, (size_t)(nbar + bsbar) * row));
    char *sx = static_cast<char *>(ctx->in_x.p), *sb = static_cast<char *>(ctx->in_xbar.p);
    const cudaMemcpyKind kind = mem == ET_HOST ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice;
    CUDA_TRY(cudaMemcpyAsync(sx, x, (size_t)n * row, kind, ctx->stream));
    CUDA_TRY(cudaMemcpyAsync(sx + (size_t)n * row, bx, (size_t)bs * row, kind, ctx->stream));
    CUDA_TRY(cudaMemcpyAsync(sb, xbar, (size_t)nbar * row, kind, ctx->stream));
    CUDA_TRY(cudaMemcpyAsync(sb + (size_t)nbar * row, bxbar, (size_t)bsbar * row, kind, ctx->stream));
    if (mem == ET_HOST) CUDA_TRY(cudaStreamSynchronize(ctx->stream));  // the caller's buffers may be pageable
    const long long cnt[4] = {n, bs, nbar, bsbar};
    layout_four(L, n + bs, nbar + bsbar, cnt);
    ET_TRY(upload_tile_classes(ctx, L));
    ET_TRY(ensure(ctx, ctx->src, (size_t)L.npad * sizeof(int)));
    PrepParams PP{};
    PP.npad = L.npad; PP.ncls = 4;
    for (int c = 0; c <= 4; ++c) PP.seg_pos[c] = L.seg_pos[c];
    for (int c = 0; c < 4; ++c) PP.seg_count[c] = L.seg_count[c];
    k_src_runs<<<ctx->num_sms * 4, 256, 0, ctx->stream>>>(PP, nullptr, static_cast<int *>(ctx->src.p));
    LAUNCH_CHECK();
    ET_TRY(run_prep(ctx, sx, sb, nullptr, nullptr, static_cast<const int *>(ctx->src.p), L, dim, dtype, sigma));
    ET_TRY(run_pairs_T(ctx, L, dim));
    ET_TRY(ensure(ctx, ctx->result, sizeof(DevPerm) + sizeof(DevT) * 4 + sizeof(DevBkg)));
    const long long Nall = n + nbar + bs + bsbar;
    k_stat_eq3<<<1, 32, 0, ctx->stream>>>(static_cast<const double *>(ctx->sums.p), (double)n, (double)nbar, (double)bs, (double)bsbar, b, bbar,
                                          Nall * (Nall - 1) / 2, static_cast<DevBkg *>(ctx->result.p), nullptr);
    LAUNCH_CHECK();
    ET_TRY(fetch(ctx, ctx->result.p, &r));
    return ET_OK;
}

et_status bkg_check(et_ctx *ctx, const void *x, int64_t n, const void *xbar, int64_t nbar, const void *bx, int64_t bs, const void *bxbar,
                    int64_t bsbar, double b, double bbar, int dim, et_dtype dtype, et_memspace mem, double sigma)
{
    ET_TRY(check_common(ctx, x, n, xbar, nbar, dim, dtype, mem, sigma));
    if (!bx || !bxbar) return fail(ctx, ET_ERR_INVALID, "null background sample");
    if (bs < 2 || bsbar < 2) return fail(ctx, ET_ERR_INVALID, "background samples need >= 2 events (Eq. 3 divides by b_s(b_s-1)); got %lld, %lld", (long long)bs, (long long)bsbar);
    if (n + nbar + bs + bsbar >= (1ll << 31)) return fail(ctx, ET_ERR_INVALID, "total number of events must be < 2^31");
    if (!(b >= 0.0) || !(bbar >= 0.0) || !std::isfinite(b) || !std::isfinite(bbar)) return fail(ctx, ET_ERR_INVALID, "b and bbar must be finite and >= 0");
    return ET_OK;
}

}  // namespace
extern "C" {

et_status et_T_bkg(et_ctx *ctx, const void *x, int64_t n, const void *xbar, int64_t nbar, const void *bx, int64_t bs,
                   const void *bxbar, int64_t bsbar, double b, double bbar, int dim, et_dtype dtype, et_memspace mem, double sigma,
                   et_bkg_result *out)
{
    ET_TRY(bkg_check(ctx, x, n, xbar, nbar, bx, bs, bxbar, bsbar, b, bbar, dim, dtype, mem, sigma));
    if (!out) return fail(ctx, ET_ERR_INVALID, "null output");
    ET_TRY(begin_call(ctx));
    Layout L;
    DevBkg r;
    ET_TRY(bkg_observed(ctx, x, n, xbar, nbar, bx, bs, bxbar, bsbar, b, bbar, dim, dtype, mem, sigma, L, r));
    ET_TRY(end_call(ctx));
    if (r.status != 0) return fail(ctx, ET_ERR_DEGENERATE, "Eq. 3 normalisation degenerate: w = n - b = %g, wbar = nbar - bbar = %g (need > 1)", r.r.w, r.r.wbar);
    *out = r.r;
    return ET_OK;
}

et_status et_bkg_permutation_test(et_ctx *ctx, const void *x, int64_t n, const void *xbar, int64_t nbar, const void *bx, int64_t bs,
                                  const void *bxbar, int64_t bsbar, double b, double bbar, int dim, et_dtype dtype, et_memspace mem,
                                  double sigma, int64_t nperm, uint64_t seed, double *T_perm, et_bkg_perm_result *out)
{
    ET_TRY(bkg_check(ctx, x, n, xbar, nbar, bx, bs, bxbar, bsbar, b, bbar, dim, dtype, mem, sigma));
    if (!out || !T_perm) return fail(ctx, ET_ERR_INVALID, "null output");
    if (nperm < 1 || nperm > ET_MAX_NPERM) return fail(ctx, ET_ERR_INVALID, "nperm must be in 1..%d", ET_MAX_NPERM);
    ET_TRY(begin_call(ctx));
    Layout L;
    DevBkg obs;
    ET_TRY(bkg_observed(ctx, x, n, xbar, nbar, bx, bs, bxbar, bsbar, b, bbar, dim, dtype, mem, sigma, L, obs));
    if (obs.status != 0) return fail(ctx, ET_ERR_DEGENERATE, "Eq. 3 normalisation degenerate: w = n - b = %g, wbar = nbar - bbar = %g (need > 1)", obs.r.w, obs.r.wbar);
    // purity of the permuted samples (reading R18): a random flavour spreads the b + bbar background events over the
    // two main samples in proportion to their sizes
    const double bp = (b + bbar) * (double)n / (double)(n + nbar), bbp = (b + bbar) * (double)nbar / (double)(n + nbar);
    if (!((double)n - bp > 1.0) || !((double)nbar - bbp > 1.0)) return fail(ctx, ET_ERR_DEGENERATE, "Eq. 3 normalisation of the permuted samples degenerate");

    // labels of both pools: select states of the n-th (bs-th) smallest composite of every permutation
    ET_TRY(span_begin(ctx, 4));
    const uint64_t seed_b = seed ^ 0x9E3779B97F4A7C15ull;
    ET_TRY(run_label_select(ctx, n + nbar, n, (int)nperm, seed));
    ET_TRY(ensure(ctx, ctx->mask, 2 * (size_t)nperm * sizeof(SelState)));
    SelState *sel_m = static_cast<SelState *>(ctx->mask.p), *sel_b = sel_m + nperm;
    CUDA_TRY(cudaMemcpyAsync(sel_m, ctx->sel.p, (size_t)nperm * sizeof(SelState), cudaMemcpyDeviceToDevice, ctx->stream));
    ET_TRY(run_label_select(ctx, bs + bsbar, bs, (int)nperm, seed_b));
    CUDA_TRY(cudaMemcpyAsync(sel_b, ctx->sel.p, (size_t)nperm * sizeof(SelState), cudaMemcpyDeviceToDevice, ctx->stream));
    ET_TRY(span_end(ctx, 4, &ctx->acc_labels_ms));

    // the identity-layout records are kept aside; every permutation gathers its own order from them
    const int F = rec_floats(dim);
    const size_t rec_bytes = (size_t)L.npad * F * sizeof(float);
    ET_TRY(ensure(ctx, ctx->recP, rec_bytes));
    CUDA_TRY(cudaMemcpyAsync(ctx->recP.p, ctx->rec.p, rec_bytes, cudaMemcpyDeviceToDevice, ctx->stream));
    k_fill_int<<<ctx->num_sms * 4, 256, 0, ctx->stream>>>(static_cast<int *>(ctx->src.p), L.npad, -1);
    LAUNCH_CHECK();
    ET_TRY(ensure(ctx, ctx->tperm, (size_t)nperm * sizeof(double)));
    BkgPermParams BP{};
    BP.n = n; BP.nbar = nbar; BP.bs = bs; BP.bsbar = bsbar;
    for (int c = 0; c < 4; ++c) BP.pos0[c] = L.seg_pos[c];
    BP.seedm_lo = (uint32_t)(seed & 0xffffffffu); BP.seedm_hi = (uint32_t)(seed >> 32);
    BP.seedb_lo = (uint32_t)(seed_b & 0xffffffffu); BP.seedb_hi = (uint32_t)(seed_b >> 32);
    DevBkg *scratch = reinterpret_cast<DevBkg *>(static_cast<char *>(ctx->result.p) + sizeof(DevPerm) + sizeof(DevT) * 4);
    const long long Nall = n + nbar + bs + bsbar;
    // per permutation: class of every source event, stable four-way partition (multi-block: k_part_*), gather, one pass
    const int nblk = (int)((Nall + kPartBlock - 1) / kPartBlock);
    ET_TRY(ensure(ctx, ctx->esccls, (size_t)Nall));
    ET_TRY(ensure(ctx, ctx->blkcnt, (size_t)nblk * 4 * sizeof(int)));
    ET_TRY(ensure(ctx, ctx->totals, 16 * sizeof(long long)));
    CUDA_TRY(cudaMemcpyAsync(static_cast<long long *>(ctx->totals.p) + 8, L.seg_pos, 4 * sizeof(long long), cudaMemcpyHostToDevice, ctx->stream));
    CUDA_TRY(cudaStreamSynchronize(ctx->stream));
    LabelOut lo{};
    lo.nseg = L.ncls;
    for (int c = 0; c <= L.ncls; ++c) lo.seg_first[c] = L.seg_first[c];
    for (int c = 0; c < L.ncls; ++c) lo.seg_pos[c] = L.seg_pos[c];
    for (int64_t p = 0; p < nperm; ++p) {
        k_bkg_class<<<(unsigned)((Nall + kThreads - 1) / kThreads), kThreads, 0, ctx->stream>>>(BP, ctx->opt_perm_offset + p, sel_m + p, sel_b + p,
                                                                                              static_cast<uint8_t *>(ctx->esccls.p));
        LAUNCH_CHECK();
        k_part_count<<<nblk, kPartBlock, 0, ctx->stream>>>(Nall, static_cast<const uint8_t *>(ctx->esccls.p), static_cast<int *>(ctx->blkcnt.p));
        LAUNCH_CHECK();
        k_part_scan<<<1, 32, 0, ctx->stream>>>(nblk, static_cast<int *>(ctx->blkcnt.p), static_cast<long long *>(ctx->totals.p));
        LAUNCH_CHECK();
        k_part_scatter<<<nblk, kPartBlock, 0, ctx->stream>>>(Nall, static_cast<const uint8_t *>(ctx->esccls.p), static_cast<const int *>(ctx->blkcnt.p),
                                                            static_cast<const long long *>(ctx->totals.p) + 8, static_cast<int *>(ctx->src.p));
        LAUNCH_CHECK();
        k_esc_gather<<<ctx->num_sms * 4, 256, 0, ctx->stream>>>(static_cast<const float4 *>(ctx->recP.p), static_cast<const int *>(ctx->src.p), L.npad,
                                                               F / 4, lo, static_cast<float4 *>(ctx->rec.p));
        LAUNCH_CHECK();
        ET_TRY(run_pairs_T(ctx, L, dim));
        k_stat_eq3<<<1, 32, 0, ctx->stream>>>(static_cast<const double *>(ctx->sums.p), (double)n, (double)nbar, (double)bs, (double)bsbar, bp, bbp,
                                              Nall * (Nall - 1) / 2, scratch, static_cast<double *>(ctx->tperm.p) + p);
        LAUNCH_CHECK();
    }
    const double guard = 1e-9 * (std::fabs(obs.r.T_xx) + std::fabs(obs.r.T_bb) + std::fabs(obs.r.T_xb));
    ET_TRY(ensure(ctx, ctx->count64, 16));
    k_count_gt<<<1, 256, 0, ctx->stream>>>(static_cast<const double *>(ctx->tperm.p), (int)nperm, obs.r.T, guard, static_cast<long long *>(ctx->count64.p));
    LAUNCH_CHECK();
    long long cnt2[2];
    ET_TRY(fetch(ctx, ctx->count64.p, &cnt2));
    CUDA_TRY(cudaMemcpyAsync(T_perm, ctx->tperm.p, (size_t)nperm * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    CUDA_TRY(cudaStreamSynchronize(ctx->stream));
    ET_TRY(end_call(ctx));
    out->observed = obs.r;
    out->count_gt = cnt2[0];
    out->n_near = cnt2[1];
    out->nperm = nperm;
    out->p_value = (double)cnt2[0] / (double)nperm;
    return ET_OK;
}

et_status et_permutation_test(et_ctx *ctx, const void *x, const double *wx, int64_t n, const void *xbar, const double *wxbar,
                              int64_t nbar, int dim, et_dtype dtype, et_memspace mem, double sigma, int64_t nperm, uint64_t seed,
                              double *T_perm, et_perm_result *out)
{
    ET_TRY(check_common(ctx, x, n, xbar, nbar, dim, dtype, mem, sigma));
    if (!out || !T_perm) return fail(ctx, ET_ERR_INVALID, "null output");
    if ((wx == nullptr) != (wxbar == nullptr)) return fail(ctx, ET_ERR_INVALID, "give both weight arrays or neither");
    if (nperm < 1 || nperm > ET_MAX_NPERM) return fail(ctx, ET_ERR_INVALID, "nperm must be in 1..%d", ET_MAX_NPERM);
    ET_TRY(begin_call(ctx));
    const void *dx = nullptr, *dxb = nullptr, *dwx = nullptr, *dwb = nullptr;
    ET_TRY(stage_in(ctx, x, (size_t)n * dim * elem_size(dtype), mem, ctx->in_x, &dx));
    ET_TRY(stage_in(ctx, xbar, (size_t)nbar * dim * elem_size(dtype), mem, ctx->in_xbar, &dxb));
    ET_TRY(stage_in(ctx, wx, (size_t)n * 8, mem, ctx->in_wx, &dwx));
    ET_TRY(stage_in(ctx, wxbar, (size_t)nbar * 8, mem, ctx->in_wxbar, &dwb));
    Layout L;
    layout_two(L, n, nbar);
    ET_TRY(upload_tile_classes(ctx, L));
    ET_TRY(run_prep(ctx, dx, dxb, static_cast<const double *>(dwx), static_cast<const double *>(dwb), nullptr, L, dim, dtype, sigma));
    et_perm_result r;
    if (use_tc(ctx, L)) {
        ET_TRY(run_perm_tc(ctx, L, dim, (int)nperm, seed, wx != nullptr, 0x1u, pairs_two(n, nbar), pairs_two(n, nbar), T_perm, &r, nullptr));
    } else {
        int nwords = 0;
        ET_TRY(run_labels_internal(ctx, L, (int)nperm, seed, &nwords));
        ET_TRY(run_pairs_rows(ctx, L, dim));
        ET_TRY(run_perm_sums(ctx, L, dim, nwords));
        ET_TRY(finish_perm(ctx, nwords, nperm, pairs_two(n, nbar), (double)n, (double)nbar, T_perm, &r));
    }
    ET_TRY(end_call(ctx));
    *out = r;
    return ET_OK;
}

et_status et_permutation_test_sigmas(et_ctx *ctx, const void *x, const double *wx, int64_t n, const void *xbar, const double *wxbar,
                                     int64_t nbar, int dim, et_dtype dtype, et_memspace mem, const double *sigmas, int nsig,
                                     int64_t nperm, uint64_t seed, double *T_perm, et_perm_result *out)
{
    if (!ctx) return ET_ERR_INVALID;
    if (!sigmas || nsig < 1 || nsig > ET_MAX_SCAN) return fail(ctx, ET_ERR_INVALID, "nsig must be in 1..%d", ET_MAX_SCAN);
    for (int s = 0; s < nsig; ++s) ET_TRY(check_common(ctx, x, n, xbar, nbar, dim, dtype, mem, sigmas[s]));
    if (!out || !T_perm) return fail(ctx, ET_ERR_INVALID, "null output");
    if ((wx == nullptr) != (wxbar == nullptr)) return fail(ctx, ET_ERR_INVALID, "give both weight arrays or neither");
    if (nperm < 1 || nperm > ET_MAX_NPERM) return fail(ctx, ET_ERR_INVALID, "nperm must be in 1..%d", ET_MAX_NPERM);
    ET_TRY(begin_call(ctx));
    const void *dx = nullptr, *dxb = nullptr, *dwx = nullptr, *dwb = nullptr;
    ET_TRY(stage_in(ctx, x, (size_t)n * dim * elem_size(dtype), mem, ctx->in_x, &dx));
    ET_TRY(stage_in(ctx, xbar, (size_t)nbar * dim * elem_size(dtype), mem, ctx->in_xbar, &dxb));
    ET_TRY(stage_in(ctx, wx, (size_t)n * 8, mem, ctx->in_wx, &dwx));
    ET_TRY(stage_in(ctx, wxbar, (size_t)nbar * 8, mem, ctx->in_wxbar, &dwb));
    Layout L;
    layout_two(L, n, nbar);
    ET_TRY(upload_tile_classes(ctx, L));
    std::vector<et_perm_result> res((size_t)nsig);
    std::vector<double> tp((size_t)nsig * (size_t)nperm);
    const bool tcpath = use_tc(ctx, L);
    int nwords = 0;
    for (int s = 0; s < nsig; ++s) {
        // the records carry the scale of sigma; the labels depend on (N, n, nperm, seed) only and are generated once
        ET_TRY(run_prep(ctx, dx, dxb, static_cast<const double *>(dwx), static_cast<const double *>(dwb), nullptr, L, dim, dtype, sigmas[s]));
        if (tcpath) {
            ET_TRY(run_perm_tc(ctx, L, dim, (int)nperm, seed, wx != nullptr, 0x1u, pairs_two(n, nbar), pairs_two(n, nbar),
                               tp.data() + (size_t)s * nperm, &res[(size_t)s], nullptr, s > 0));
        } else {
            if (s == 0) ET_TRY(run_labels_internal(ctx, L, (int)nperm, seed, &nwords));
            ET_TRY(run_pairs_rows(ctx, L, dim));
            ET_TRY(run_perm_sums(ctx, L, dim, nwords));
            ET_TRY(finish_perm(ctx, nwords, nperm, pairs_two(n, nbar), (double)n, (double)nbar, tp.data() + (size_t)s * nperm, &res[(size_t)s]));
        }
    }
    ET_TRY(end_call(ctx));
    memcpy(T_perm, tp.data(), tp.size() * sizeof(double));
    for (int s = 0; s < nsig; ++s) out[s] = res[(size_t)s];
    return ET_OK;
}

et_status et_podd_split(et_ctx *ctx, const double *pB, const double *pC, const double *pD, int64_t n, int is_conjugate,
                        et_memspace mem, uint8_t *positive, int64_t *n_positive)
{
    if (!ctx) return ET_ERR_INVALID;
    if (!pB || !pC || !pD || !positive || n < 1) return fail(ctx, ET_ERR_INVALID, "null pointer or n < 1");
    ET_TRY(begin_call(ctx));
    const void *dB, *dC, *dD;
    ET_TRY(stage_in(ctx, pB, (size_t)n * 24, mem, ctx->in_mx, &dB));
    ET_TRY(stage_in(ctx, pC, (size_t)n * 24, mem, ctx->in_mb, &dC));
    ET_TRY(stage_in(ctx, pD, (size_t)n * 24, mem, ctx->in_aux, &dD));
    uint8_t *dpos = positive;
    if (mem == ET_HOST) { ET_TRY(ensure(ctx, ctx->posx, (size_t)n)); dpos = static_cast<uint8_t *>(ctx->posx.p); }
    ET_TRY(ensure(ctx, ctx->count64, 8));
    CUDA_TRY(cudaMemsetAsync(ctx->count64.p, 0, 8, ctx->stream));
    k_podd_flags<<<(unsigned)((n + 255) / 256), 256, 0, ctx->stream>>>(static_cast<const double *>(dB), static_cast<const double *>(dC),
                                                                    static_cast<const double *>(dD), n, 3, is_conjugate, dpos,
                                                                    static_cast<unsigned long long *>(ctx->count64.p));
    LAUNCH_CHECK();
    if (mem == ET_HOST) CUDA_TRY(cudaMemcpyAsync(positive, dpos, (size_t)n, cudaMemcpyDeviceToHost, ctx->stream));
    unsigned long long cnt = 0;
    ET_TRY(fetch(ctx, ctx->count64.p, &cnt));
    ET_TRY(end_call(ctx));
    if (n_positive) *n_positive = (int64_t)cnt;
    return ET_OK;
}

et_status et_podd_test(et_ctx *ctx, const void *x, const double *mom_x, int64_t n, const void *xbar, const double *mom_xbar,
                       int64_t nbar, int dim, et_dtype dtype, et_memspace mem, double sigma, int64_t nperm, uint64_t seed,
                       double *T_perm, et_podd_result *out)
{
    ET_TRY(check_common(ctx, x, n, xbar, nbar, dim, dtype, mem, sigma));
    if (!out || !T_perm || !mom_x || !mom_xbar) return fail(ctx, ET_ERR_INVALID, "null pointer");
    if (nperm < 1 || nperm > ET_MAX_NPERM) return fail(ctx, ET_ERR_INVALID, "nperm must be in 1..%d", ET_MAX_NPERM);
    ET_TRY(begin_call(ctx));
    const void *dx = nullptr, *dxb = nullptr, *dmx = nullptr, *dmb = nullptr;
    ET_TRY(stage_in(ctx, x, (size_t)n * dim * elem_size(dtype), mem, ctx->in_x, &dx));
    ET_TRY(stage_in(ctx, xbar, (size_t)nbar * dim * elem_size(dtype), mem, ctx->in_xbar, &dxb));
    ET_TRY(stage_in(ctx, mom_x, (size_t)n * 72, mem, ctx->in_mx, &dmx));
    ET_TRY(stage_in(ctx, mom_xbar, (size_t)nbar * 72, mem, ctx->in_mb, &dmb));
    const long long N = n + nbar;

    // H0: the split (Eq. 4) and the stable partition into the layout classes (I, IV | II, III)
    ET_TRY(ensure(ctx, ctx->posx, (size_t)n));
    ET_TRY(ensure(ctx, ctx->posb, (size_t)nbar));
    ET_TRY(ensure(ctx, ctx->count64, 16));
    CUDA_TRY(cudaMemsetAsync(ctx->count64.p, 0, 16, ctx->stream));
    const double *mx = static_cast<const double *>(dmx), *mb = static_cast<const double *>(dmb);
    k_podd_flags<<<(unsigned)((n + 255) / 256), 256, 0, ctx->stream>>>(mx, mx + 3, mx + 6, n, 9, 0, static_cast<uint8_t *>(ctx->posx.p),
                                                                    static_cast<unsigned long long *>(ctx->count64.p));
    LAUNCH_CHECK();
    k_podd_flags<<<(unsigned)((nbar + 255) / 256), 256, 0, ctx->stream>>>(mb, mb + 3, mb + 6, nbar, 9, 1, static_cast<uint8_t *>(ctx->posb.p),
                                                                       static_cast<unsigned long long *>(ctx->count64.p) + 1);
    LAUNCH_CHECK();
    unsigned long long pos_cnt[2];
    ET_TRY(fetch(ctx, ctx->count64.p, &pos_cnt));
    const long long nI = (long long)pos_cnt[0], nII = n - nI, nIII = (long long)pos_cnt[1], nIV = nbar - nIII;
    const long long cnt[4] = {nI, nIV, nII, nIII};  // layout order
    if (nI + nIV < 2 || nII + nIII < 2) return fail(ctx, ET_ERR_INVALID, "P-odd samples need >= 2 events each (I+IV = %lld, II+III = %lld)", nI + nIV, nII + nIII);
    Layout L;
    layout_four(L, n, nbar, cnt);
    ET_TRY(upload_tile_classes(ctx, L));
    const int nblk = (int)((N + kPartBlock - 1) / kPartBlock);
    ET_TRY(ensure(ctx, ctx->blkcnt, (size_t)nblk * 4 * sizeof(int)));
    ET_TRY(ensure(ctx, ctx->totals, 16 * sizeof(long long)));
    ET_TRY(ensure(ctx, ctx->src, (size_t)L.npad * sizeof(int)));
    k_fill_int<<<ctx->num_sms * 4, 256, 0, ctx->stream>>>(static_cast<int *>(ctx->src.p), L.npad, -1);
    LAUNCH_CHECK();
    ET_TRY(ensure(ctx, ctx->esccls, (size_t)N));
    k_podd_classes<<<(unsigned)((N + 255) / 256), 256, 0, ctx->stream>>>(N, n, static_cast<const uint8_t *>(ctx->posx.p),
                                                                      static_cast<const uint8_t *>(ctx->posb.p),
                                                                      static_cast<uint8_t *>(ctx->esccls.p));
    LAUNCH_CHECK();
    k_part_count<<<nblk, kPartBlock, 0, ctx->stream>>>(N, static_cast<const uint8_t *>(ctx->esccls.p), static_cast<int *>(ctx->blkcnt.p));
    LAUNCH_CHECK();
    k_part_scan<<<1, 32, 0, ctx->stream>>>(nblk, static_cast<int *>(ctx->blkcnt.p), static_cast<long long *>(ctx->totals.p));
    LAUNCH_CHECK();
    CUDA_TRY(cudaMemcpyAsync(static_cast<long long *>(ctx->totals.p) + 8, L.seg_pos, 4 * sizeof(long long), cudaMemcpyHostToDevice, ctx->stream));
    k_part_scatter<<<nblk, kPartBlock, 0, ctx->stream>>>(N, static_cast<const uint8_t *>(ctx->esccls.p),
                                                        static_cast<const int *>(ctx->blkcnt.p), static_cast<const long long *>(ctx->totals.p) + 8,
                                                        static_cast<int *>(ctx->src.p));
    LAUNCH_CHECK();

    ET_TRY(run_prep(ctx, dx, dxb, nullptr, nullptr, static_cast<const int *>(ctx->src.p), L, dim, dtype, sigma));
    if (use_tc(ctx, L)) {
        // layout classes: 0 = I, 1 = IV, 2 = II, 3 = III; P-even sample X = I + II = classes {0, 2}
        et_perm_result pr;
        et_result even;
        ET_TRY(run_perm_tc(ctx, L, dim, (int)nperm, seed, false, 0x5u, pairs_two(nI + nIV, nII + nIII), pairs_two(n, nbar), T_perm, &pr, &even));
        ET_TRY(end_call(ctx));
        out->count[0] = nI; out->count[1] = nII; out->count[2] = nIII; out->count[3] = nIV;
        out->p_even = even;
        out->p_odd = pr;
        return ET_OK;
    }
    ET_TRY(run_class_weights(ctx, L, dim));
    int nwords = 0;
    ET_TRY(run_labels_internal(ctx, L, (int)nperm, seed, &nwords));
    ET_TRY(run_pairs_rows(ctx, L, dim));

    // P-even T of (I+II) vs (III+IV) from the class-pair sums of the same pass: layout classes {0 (I), 2 (II)} = X
    const int nt = (int)(L.npad / kPad);
    ET_TRY(ensure(ctx, ctx->clssum, (size_t)nt * 4 * sizeof(double)));
    ET_TRY(ensure(ctx, ctx->sums, 2 * kSumSlots * sizeof(double)));
    k_class_sums<4><<<nt, kThreads, 0, ctx->stream>>>(static_cast<const float *>(ctx->rec.p), rec_floats(dim), dim,
                                                     static_cast<const double *>(ctx->rowsum.p), L.npad, static_cast<double *>(ctx->clssum.p));
    LAUNCH_CHECK();
    double *M = static_cast<double *>(ctx->sums.p) + kSumSlots;
    CUDA_TRY(cudaMemsetAsync(M, 0, kSumSlots * sizeof(double), ctx->stream));
    k_reduce_by_class<<<1, 16, 0, ctx->stream>>>(static_cast<const double *>(ctx->clssum.p), static_cast<const uint8_t *>(ctx->tilecls.p), nt, 4, M);
    LAUNCH_CHECK();
    k_sym_class_sums<<<1, 32, 0, ctx->stream>>>(M, 4, static_cast<double *>(ctx->sums.p));
    LAUNCH_CHECK();
    ET_TRY(ensure(ctx, ctx->result, sizeof(DevPerm) + sizeof(DevT) * 4));
    DevT *dev_even = reinterpret_cast<DevT *>(static_cast<char *>(ctx->result.p) + sizeof(DevPerm));
    k_stat_from_sums<<<1, 32, 0, ctx->stream>>>(static_cast<const double *>(ctx->sums.p), static_cast<const double *>(ctx->clsw.p), 4,
                                                0x5u, pairs_two(n, nbar), dev_even);
    LAUNCH_CHECK();

    ET_TRY(run_perm_sums(ctx, L, dim, nwords));
    et_perm_result pr;
    ET_TRY(finish_perm(ctx, nwords, nperm, pairs_two(nI + nIV, nII + nIII), (double)(nI + nIV), (double)(nII + nIII), T_perm, &pr));
    DevT even;
    ET_TRY(fetch(ctx, dev_even, &even));
    ET_TRY(end_call(ctx));
    out->count[0] = nI; out->count[1] = nII; out->count[2] = nIII; out->count[3] = nIV;
    out->p_even = even.r;
    out->p_odd = pr;
    return ET_OK;
}

et_status et_perm_labels(et_ctx *ctx, int64_t N, int64_t n, int64_t nperm, uint64_t seed, et_memspace mem, uint32_t *mask)
{
    if (!ctx) return ET_ERR_INVALID;
    if (!mask || N < 1 || n < 1 || n > N || N >= (1ll << 31)) return fail(ctx, ET_ERR_INVALID, "bad label arguments");
    if (nperm < 1 || nperm > ET_MAX_NPERM) return fail(ctx, ET_ERR_INVALID, "nperm must be in 1..%d", ET_MAX_NPERM);
    ET_TRY(begin_call(ctx));
    ET_TRY(span_begin(ctx, 4));
    ET_TRY(run_label_select(ctx, N, n, (int)nperm, seed));
    const int nwords = (int)((nperm + 31) / 32);
    uint32_t *dmask = mask;
    const size_t bytes = (size_t)N * nwords * sizeof(uint32_t);
    if (mem == ET_HOST) { ET_TRY(ensure(ctx, ctx->mask, bytes)); dmask = static_cast<uint32_t *>(ctx->mask.p); }
    LabelOut lo{};
    lo.stride_g = 1;
    lo.stride_i = nwords;
    lo.nseg = 0;
    const dim3 grid((unsigned)((N + kThreads - 1) / kThreads), (unsigned)nwords);
    k_label_write<<<grid, kThreads, 0, ctx->stream>>>(N, n, (int)nperm, ctx->opt_perm_offset, 0, nwords, (uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32),
                                                     static_cast<const SelState *>(ctx->sel.p), lo, dmask);
    LAUNCH_CHECK();
    ET_TRY(span_end(ctx, 4, &ctx->acc_labels_ms));
    if (mem == ET_HOST) CUDA_TRY(cudaMemcpyAsync(mask, dmask, bytes, cudaMemcpyDeviceToHost, ctx->stream));
    ET_TRY(end_call(ctx));
    return ET_OK;
}

et_status et_row_sums(et_ctx *ctx, const void *x, const double *wx, int64_t n, const void *xbar, const double *wxbar, int64_t nbar,
                      int dim, et_dtype dtype, et_memspace mem, double sigma, const int64_t *rows, int64_t nrows, double *r_x,
                      double *r_xbar)
{
    ET_TRY(check_common(ctx, x, n, xbar, nbar, dim, dtype, mem, sigma));
    if (!rows || !r_x || !r_xbar || nrows < 1) return fail(ctx, ET_ERR_INVALID, "null pointer or nrows < 1");
    if ((wx == nullptr) != (wxbar == nullptr)) return fail(ctx, ET_ERR_INVALID, "give both weight arrays or neither");
    for (int64_t k = 0; k < nrows; ++k)
        if (rows[k] < 0 || rows[k] >= n + nbar) return fail(ctx, ET_ERR_INVALID, "row index out of range");
    ET_TRY(begin_call(ctx));
    const void *dx = nullptr, *dxb = nullptr, *dwx = nullptr, *dwb = nullptr;
    ET_TRY(stage_in(ctx, x, (size_t)n * dim * elem_size(dtype), mem, ctx->in_x, &dx));
    ET_TRY(stage_in(ctx, xbar, (size_t)nbar * dim * elem_size(dtype), mem, ctx->in_xbar, &dxb));
    ET_TRY(stage_in(ctx, wx, (size_t)n * 8, mem, ctx->in_wx, &dwx));
    ET_TRY(stage_in(ctx, wxbar, (size_t)nbar * 8, mem, ctx->in_wxbar, &dwb));
    Layout L;
    layout_two(L, n, nbar);
    ET_TRY(upload_tile_classes(ctx, L));
    ET_TRY(run_prep(ctx, dx, dxb, static_cast<const double *>(dwx), static_cast<const double *>(dwb), nullptr, L, dim, dtype, sigma));
    ET_TRY(run_pairs_rows(ctx, L, dim, false));
    std::vector<long long> pos((size_t)nrows);
    for (int64_t k = 0; k < nrows; ++k) pos[(size_t)k] = rows[k] < n ? rows[k] : L.seg_pos[1] + (rows[k] - n);
    ET_TRY(ensure(ctx, ctx->rows, (size_t)nrows * 8));
    ET_TRY(ensure(ctx, ctx->rowsout, (size_t)nrows * 16));
    CUDA_TRY(cudaMemcpyAsync(ctx->rows.p, pos.data(), (size_t)nrows * 8, cudaMemcpyHostToDevice, ctx->stream));
    k_gather_rows<<<(unsigned)((nrows + 255) / 256), 256, 0, ctx->stream>>>(static_cast<const double *>(ctx->rowsum.p), L.npad,
                                                                         static_cast<const long long *>(ctx->rows.p), nrows, 2,
                                                                         static_cast<double *>(ctx->rowsout.p));
    LAUNCH_CHECK();
    CUDA_TRY(cudaMemcpyAsync(r_x, ctx->rowsout.p, (size_t)nrows * 8, cudaMemcpyDeviceToHost, ctx->stream));
    CUDA_TRY(cudaMemcpyAsync(r_xbar, static_cast<double *>(ctx->rowsout.p) + nrows, (size_t)nrows * 8, cudaMemcpyDeviceToHost, ctx->stream));
    ET_TRY(end_call(ctx));
    return ET_OK;
}

et_status et_scp(et_ctx *ctx, const void *x, int64_t n, const void *xbar, int64_t nbar, int dim, et_dtype dtype, et_memspace mem,
                 const double *lo, const double *hi, const int32_t *nbins, double *S, int64_t *Nx, int64_t *Nxbar, et_scp_result *out)
{
    if (!ctx) return ET_ERR_INVALID;
    if (!x || !xbar || !lo || !hi || !nbins || !out) return fail(ctx, ET_ERR_INVALID, "null pointer");
    if (n < 1 || nbar < 1) return fail(ctx, ET_ERR_INVALID, "n and nbar must be >= 1");
    if (dim < 1 || dim > scp::kMaxAxes) return fail(ctx, ET_ERR_INVALID, "dim must be in 1..%d; got %d", scp::kMaxAxes, dim);
    if (dtype != ET_F32 && dtype != ET_F64) return fail(ctx, ET_ERR_INVALID, "bad dtype");
    if (mem != ET_HOST && mem != ET_DEVICE) return fail(ctx, ET_ERR_INVALID, "bad memspace");
    scp::Grid G{};
    G.dim = dim;
    long long total = 1;
    for (int k = 0; k < dim; ++k) {
        if (!std::isfinite(lo[k]) || !std::isfinite(hi[k]) || !(lo[k] < hi[k])) return fail(ctx, ET_ERR_INVALID, "axis %d: need finite lo < hi", k);
        if (nbins[k] < 1) return fail(ctx, ET_ERR_INVALID, "axis %d: nbins must be >= 1", k);
        G.lo[k] = lo[k]; G.hi[k] = hi[k]; G.nbins[k] = nbins[k];
        total *= nbins[k];
        if (total > scp::kMaxBins) return fail(ctx, ET_ERR_INVALID, "more than 2^24 bins");
    }
    G.total = (int)total;
    ET_TRY(begin_call(ctx));
    const void *dx = nullptr, *dxb = nullptr;
    ET_TRY(stage_in(ctx, x, (size_t)n * dim * elem_size(dtype), mem, ctx->in_x, &dx));
    ET_TRY(stage_in(ctx, xbar, (size_t)nbar * dim * elem_size(dtype), mem, ctx->in_xbar, &dxb));
    // counts: [Nx total][Nxbar total][outside 1]
    const size_t cnt_bytes = (2 * (size_t)total + 1) * sizeof(unsigned long long);
    ET_TRY(ensure(ctx, ctx->scpcnt, cnt_bytes));
    ET_TRY(ensure(ctx, ctx->scpS, (size_t)total * sizeof(double)));
    ET_TRY(ensure(ctx, ctx->result, sizeof(scp::DevScp)));
    CUDA_TRY(cudaMemsetAsync(ctx->scpcnt.p, 0, cnt_bytes, ctx->stream));
    unsigned long long *cx = static_cast<unsigned long long *>(ctx->scpcnt.p), *cb = cx + total, *coutside = cx + 2 * total;
    const int grid = ctx->num_sms * 8;
    const bool sm = total <= scp::kSmemBins;
    auto hist = [&](const void *p, long long cnt, unsigned long long *dst) {
        const int g = (int)std::min<long long>(grid, (cnt + 255) / 256);
        if (dtype == ET_F32) {
            if (sm) scp::k_scp_hist<float, true><<<g, 256, 0, ctx->stream>>>(static_cast<const float *>(p), cnt, G, dst, coutside);
            else scp::k_scp_hist<float, false><<<g, 256, 0, ctx->stream>>>(static_cast<const float *>(p), cnt, G, dst, coutside);
        } else {
            if (sm) scp::k_scp_hist<double, true><<<g, 256, 0, ctx->stream>>>(static_cast<const double *>(p), cnt, G, dst, coutside);
            else scp::k_scp_hist<double, false><<<g, 256, 0, ctx->stream>>>(static_cast<const double *>(p), cnt, G, dst, coutside);
        }
    };
    hist(dx, n, cx);
    LAUNCH_CHECK();
    hist(dxb, nbar, cb);
    LAUNCH_CHECK();
    scp::k_scp_stat<<<1, 1024, 0, ctx->stream>>>(cx, cb, G.total, static_cast<double *>(ctx->scpS.p), static_cast<scp::DevScp *>(ctx->result.p));
    LAUNCH_CHECK();
    scp::DevScp r;
    ET_TRY(fetch(ctx, ctx->result.p, &r));
    unsigned long long n_out = 0;
    CUDA_TRY(cudaMemcpyAsync(&n_out, coutside, sizeof(n_out), cudaMemcpyDeviceToHost, ctx->stream));
    CUDA_TRY(cudaStreamSynchronize(ctx->stream));
    if (r.n_in_x < 1 || r.n_in_xbar < 1 || r.bins_used < 2) {
        ET_TRY(end_call(ctx));
        return fail(ctx, ET_ERR_DEGENERATE, "S_CP needs events of both samples inside the grid and two bins with entries (in-grid %lld, %lld; bins %lld)",
                    r.n_in_x, r.n_in_xbar, r.bins_used);
    }
    static_assert(sizeof(unsigned long long) == sizeof(int64_t), "counts are copied out as int64");
    if (S) CUDA_TRY(cudaMemcpyAsync(S, ctx->scpS.p, (size_t)total * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    if (Nx) CUDA_TRY(cudaMemcpyAsync(Nx, cx, (size_t)total * sizeof(int64_t), cudaMemcpyDeviceToHost, ctx->stream));
    if (Nxbar) CUDA_TRY(cudaMemcpyAsync(Nxbar, cb, (size_t)total * sizeof(int64_t), cudaMemcpyDeviceToHost, ctx->stream));
    ET_TRY(end_call(ctx));
    out->chi2 = r.chi2;
    out->ndf = r.bins_used - 1;
    out->p_value = scp::chi2_sf(r.chi2, r.bins_used - 1);
    out->alpha = r.alpha;
    out->n_in_x = r.n_in_x;
    out->n_in_xbar = r.n_in_xbar;
    out->n_outside = (int64_t)n_out;
    out->bins_used = r.bins_used;
    out->bins_total = total;
    return ET_OK;
}

}  // extern "C"
