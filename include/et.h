/*
 * et.h -- C ABI of libet.so: the energy-test hot path of arXiv:1612.04705 on
 * one NVIDIA B200 (sm_100a).  Citations are /root/reference/PAPER.md:<line>.
 *
 * What the library computes
 *   psi_ij = exp(-d_ij^2 / (2 sigma^2)), d_ij the Euclidean distance of events
 *   i and j in the caller's phase-space coordinates;
 *   T = sum_{i<j in X} psi/(n(n-1)) + sum_{i<j in Xbar} psi/(nbar(nbar-1))
 *       - sum_{i in X, j in Xbar} psi/(n nbar)                    (Eq. 2);
 *   its per-event-weighted form (Sect. 3; reading R7);
 *   the permutation p-value: fraction of permutation T values greater than the
 *   observed T; the Sect. 5 sample split by the sign of a triple
 *   product and the P-odd test (I+IV) vs (II+III).
 *
 * Conventions (all entry points)
 *   - Coordinates are row-major [n][dim], dtype per `et_dtype`; weights and
 *     momenta are always double.  `mem` says where EVERY array argument of the
 *     call lives except those documented as host: ET_HOST (plain host memory;
 *     the library stages it to the device itself) or ET_DEVICE (device pointers
 *     on the context's device, e.g. from PyTorch).  Inputs are never modified
 *     and never freed by the library.
 *   - Result structs and T_perm are HOST memory owned by the caller.
 *   - Pooled event index: X events are 0..n-1, Xbar events n..n+nbar-1.
 *   - The context owns a stream (or borrows the caller's), all scratch and the
 *     label buffers; it is not thread-safe (one context per host thread).
 *   - Every call is complete (stream-synchronised) on return.
 *   - ET_DEVICE inputs must be complete before the call as seen from the context's stream: produced on
 *     that stream (pass it to et_create), or synchronised by the caller (a library-owned stream is
 *     non-blocking and does not wait for the legacy default stream).  They must live on the context's device.
 *   - On any status != ET_OK the outputs are untouched and et_last_error()
 *     explains.  There is no CPU fallback: without a CUDA device et_create
 *     fails with ET_ERR_CUDA.
 *   - Limits: 1 <= dim <= ET_MAX_DIM, n >= 2, nbar >= 2, n + nbar < 2^31,
 *     1 <= nperm <= ET_MAX_NPERM.
 */
#ifndef ET_H_
#define ET_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ET_MAX_DIM 8
#define ET_MAX_NPERM 65536

typedef struct et_ctx et_ctx; /* opaque */

typedef enum {
    ET_OK = 0,
    ET_ERR_INVALID = -1,    /* null pointer, n < 2, nbar < 2, dim out of range, nperm out of range */
    ET_ERR_SIGMA = -2,      /* sigma <= 0 or not finite                                            */
    ET_ERR_NONFINITE = -3,  /* NaN/Inf in coordinates or weights (checked on the device in prep)   */
    ET_ERR_DEGENERATE = -4, /* weighted: W <= 1 or Wbar <= 1 for the observed split                */
    ET_ERR_NOMEM = -5,
    ET_ERR_CUDA = -6
} et_status;

typedef enum { ET_F32 = 0, ET_F64 = 1 } et_dtype;
typedef enum { ET_HOST = 0, ET_DEVICE = 1 } et_memspace;

/* T and its parts, in the order of Eq. 2: T = T_xx + T_bb - T_xb. */
typedef struct {
    double T, T_xx, T_bb, T_xb; /* normalised terms                                              */
    double S_xx, S_bb, S_xb;    /* raw psi sums (i<j within, all pairs across), weighted if any  */
    double W, Wbar;             /* n, nbar, or the weight sums                                   */
    int64_t n_pairs;            /* unordered pairs that enter T                                  */
} et_result;

typedef struct {
    et_result observed;
    double p_value;   /* count_gt / nperm  (strict >; reading R3)                   */
    int64_t count_gt; /* #{p : T_p > T_obs}                                                       */
    int64_t n_near;   /* permutations whose side of T_obs the arithmetic cannot certify (R5, R10):
                         #{p : |T_p - T_obs| <= guard} or T_p NaN, guard = 8 sigma of the error model
                         of T_p - T_obs (fp32 psi; on the tensor-core path
                         also the 15-bit rounding).  With ET_OPT_EXACT_P (default on) the
                         tensor-core path re-evaluates the permutations inside its band in the
                         fp32-pair / fp64-sum arithmetic of et_T and n_near is what is left after
                         that.  count_gt equals the oracle's count when n_near = 0             */
    int64_t nperm;
} et_perm_result;

typedef struct {
    int64_t count[4];    /* N(I), N(II), N(III), N(IV) of Eq. 4               */
    et_result p_even;    /* (I+II) vs (III+IV): the default X vs Xbar test        */
    et_perm_result p_odd;/* (I+IV) vs (II+III) with its permutation p-value       */
} et_podd_result;

/* Device-side timings of the last call, CUDA events on the context's stream. */
typedef struct {
    double ms_total;   /* whole call on the device, staging copies included                      */
    double ms_pairs;   /* the O(N^2) kernels only (all-pairs, row sums, permutation sums)         */
    double ms_labels;  /* permutation label generation                                            */
    int64_t launches;  /* kernels launched by the call                                            */
    int64_t pair_evals;/* psi evaluations the kernels performed (padding and diagonals included)  */
    /* the O(N^2) kernel class with the largest device time in the call (bench.py's roofline object)   */
    double ms_dominant;        /* summed device time of its launches                               */
    int64_t dominant_launches;
    int64_t dominant_ops;      /* ALGORITHMIC work of those launches: FP32-pipe thread instructions
                                  (CUDA-core kernels: unique pairs x (2 dim + 1), per mask word
                                  unique pairs x (2 dim + 32)) or 2 x MACs (tensor-core kernel; with
                                  ET_OPT_TC_SKIP in force: of the K blocks that were evaluated)       */
    char dominant_kernel[32];  /* "k_pairs_T", "k_pairs_rows", "k_perm32", "k_perm_tc" or ""       */
    int64_t dominant_ops_executed; /* k_perm_tc: the same count over the label columns the launches
                                  carried (256 or 512 per launch, the three special columns in every
                                  launch); 0 for the other kernels                                  */
    double ms_escalation;      /* device time of the guard-band escalation (ET_OPT_EXACT_P)         */
    int64_t n_near_before;     /* n_near of the tensor-core pass, before the escalation             */
    int64_t n_escalated;       /* permutations re-evaluated by the escalation                       */
    int64_t distance_form;     /* ET_OPT_DISTANCE value the last all-pairs (k_pairs_T) launch of the
                                  call ran with: 1 or 2; 0 if the call had none                      */
} et_stats;

/* Options for et_set_option. */
typedef enum {
    ET_OPT_PERM_KERNEL = 0, /* permutation sums: 0 (default) = tensor-core contraction (tcgen05
                               kind::i8, psi quantised to 15 bits, exact integer sums) when the
                               padded pooled size is >= 8192 rows, else the fp32 CUDA-core
                               kernel; 1 = always CUDA cores; 2 = always tensor cores (below
                               8192 rows the 15-bit rounding noise can exceed the 1e-6 tolerance
                               of T: a test hook)                       */
    ET_OPT_PERM_OFFSET = 1, /* first permutation index p0 (default 0): the calls evaluate
                               permutations p0 .. p0+nperm-1 of the seed's stream, T_perm[k] is
                               permutation p0+k.  Permutation p depends only on (seed, p), so
                               disjoint ranges on several GPUs / calls form one test
                               (PAPER.md:219 farms permutations out the same way).
                               p0 + nperm must stay below 2^34                                    */
    ET_OPT_EXACT_P = 2,     /* guard-band escalation of the tensor-core path: re-evaluate up to this
                               many permutations (default 16, at most 64; 0 = off) whose T_p lies
                               inside the guard band of T_obs, one 5/8 all-pairs pass each on the
                               CUDA cores (a full pass when weighted); skipped when more are inside  */
    ET_OPT_DISTANCE = 3,    /* distance arithmetic of the all-pairs kernel of et_T / et_T_weighted /
                               et_T_bkg and of the escalation: 1 = differences, e = sum_k (u_ik - u_jk)^2
                               (2 dim + 1 FP32 operations per pair); 2 = Gram form, e = |u_i|^2 +
                               |u_j|^2 - 2 u_i.u_j (dim + 2 operations; psi then carries a relative
                               rounding error of about 8e-8 |u|^2_max, |u|^2_max the squared half
                               diagonal of the bounding box over 2 sigma^2 / log2 e); 0 (default) =
                               Gram form when dim >= 4, n + nbar >= 4096 and |u|^2_max <= 48, else differences;
                               2 falls back to differences when |u|^2_max > 96 (et_stats.distance_form tells)
                               (DESIGN.md section 6).  T stays within the 1e-6 tolerance either way    */
    ET_OPT_TC_ORDER = 5,    /* row order of the tensor-core contraction: 1 (default) = the records of every class
                               segment in Morton order of their coordinates (a sorted copy; labels written
                               through the inverse map), 0 = the layout order.  The integer sums of the
                               unweighted contraction do not depend on it bit for bit (weighted sums: in
                               the last bits, far inside the guard band; the keys come from the input
                               coordinates, so a sigma scan and its single calls still agree exactly), the
                               time does: the board runs at its power cap and similar neighbouring rows
                               cost the tensor pipe less energy (-2.3 % per launch at BASELINE config 4)  */
    ET_OPT_TC_SKIP = 6,     /* exact skipping of far K blocks in the tensor-core contraction (needs ET_OPT_TC_ORDER):
                               1 (default) = (row tile, K block) pairs whose bounding boxes are farther apart than
                               the distance at which the 15-bit psi rounds to 0 (4.7 sigma) are not evaluated,
                               when that is at least 5 % of the blocks; 0 = every block.  Same sums bit for bit   */
    ET_OPT_LABEL_SELECT = 4 /* radix select of the n-th smallest composite key of every permutation
                               (reading R4): 0 (default) = four histogram sweeps over the key32 half, then
                               one sweep that lists the wanted bucket's events; 1 = eight histogram sweeps
                               (the fallback of 0 for a bucket of more than 64 events, selectable so that it
                               can be tested).  The labels are the same bits either way                    */
} et_option;

/* Create a context on CUDA device `device`.  `cuda_stream` is a cudaStream_t to
 * borrow, or NULL for a library-owned stream. */
et_status et_create(et_ctx **ctx, int device, void *cuda_stream);
void et_destroy(et_ctx *ctx);
/* Context-owned explanation of the last non-OK status; never freed by the caller. */
const char *et_last_error(const et_ctx *ctx);
et_status et_set_option(et_ctx *ctx, et_option opt, int64_t value);

/* Unit-range shard over `world` contexts (one per GPU / process): the context evaluates
 * every world-th work unit of the O(N^2) kernels (the tile-pair list of et_T, the unit table of the tensor-core
 * permutation sums) and completes its partial sums -- exact int64 column sums when unweighted, doubles otherwise --
 * through `fn`: buf is HOST memory [world][bytes_per_rank] with slice `rank` filled in; fn must return 0 with every
 * slice filled with that rank's bytes (an all-gather, e.g. over NCCL or gloo; the binding supplies one on
 * torch.distributed).  The slices are summed in rank order on the device, so all ranks return identical results;
 * unweighted results do not depend on `world` at all (integer sums).  Labels, prep and the O(N) kernels are
 * replicated; every rank must make the same calls with the same arguments.  world = 1 (fn may be NULL) switches the
 * shard off.  The small-N CUDA-core permutation kernels are not sharded (every rank evaluates them in full). */
typedef int (*et_allgather_fn)(void *user, void *buf, int64_t bytes_per_rank);
et_status et_set_shard(et_ctx *ctx, int rank, int world, et_allgather_fn fn, void *user);
et_status et_get_stats(const et_ctx *ctx, et_stats *out);
const char *et_version(void);

/* Eq. 2 for samples x[n][dim], xbar[nbar][dim]. */
et_status et_T(et_ctx *ctx, const void *x, int64_t n, const void *xbar, int64_t nbar,
               int dim, et_dtype dtype, et_memspace mem, double sigma, et_result *out);

/* Per-event-weighted Eq. 2 (reading R7): psi_ij -> w_i w_j psi_ij,
 * n -> W = sum of weights.  wx[n], wxbar[nbar] double, same memory space. */
et_status et_T_weighted(et_ctx *ctx, const void *x, const double *wx, int64_t n,
                        const void *xbar, const double *wxbar, int64_t nbar,
                        int dim, et_dtype dtype, et_memspace mem, double sigma, et_result *out);

/* Permutation test.  Permutation p reassigns the pooled events
 * to samples of the original sizes by the rule of reading R4 (Philox4x32-10
 * keys, the n smallest composites go to X); weights (both NULL or both given)
 * travel with their events.  T_perm[nperm] (host) receives the
 * permutation T values; a degenerate weighted split gives NaN and is not
 * counted.  The observed T goes through the same kernels as the T_p. */
et_status et_permutation_test(et_ctx *ctx, const void *x, const double *wx, int64_t n,
                              const void *xbar, const double *wxbar, int64_t nbar,
                              int dim, et_dtype dtype, et_memspace mem, double sigma,
                              int64_t nperm, uint64_t seed, double *T_perm, et_perm_result *out);

/* The permutation test at nsig <= ET_MAX_SCAN values of sigma: the sigma scan of Sect. 2.2 (Fig. 2
 * shows "p-values versus sigma"; BASELINE configs[1] and [3] quote three sigma x 1000 permutations).  Results are those
 * of nsig et_permutation_test calls with the same (nperm, seed) -- the same permutations serve every sigma -- bit for
 * bit; the staging copies, the permutation labels (radix select + label matrix) and the layout are made once.
 * T_perm[nsig][nperm] and out[nsig] are HOST memory. */
#define ET_MAX_SCAN 16
et_status et_permutation_test_sigmas(et_ctx *ctx, const void *x, const double *wx, int64_t n,
                                     const void *xbar, const double *wxbar, int64_t nbar,
                                     int dim, et_dtype dtype, et_memspace mem,
                                     const double *sigmas, int nsig, int64_t nperm, uint64_t seed,
                                     double *T_perm, et_perm_result *out);

/* Sect. 5 split (Eq. 4): C = pB . (pC x pD), momenta [n][3]
 * double in the mother rest frame.  positive[i] = 1 iff C > 0 (is_conjugate = 0)
 * or -C > 0 (is_conjugate = 1, momenta of the C-conjugate particles); C == 0 is
 * negative (reading R11).  `positive` lives in `mem`; *n_positive is host. */
et_status et_podd_split(et_ctx *ctx, const double *pB, const double *pC, const double *pD,
                        int64_t n, int is_conjugate, et_memspace mem,
                        uint8_t *positive, int64_t *n_positive);

/* P-odd test: split X by C_T and Xbar by -Cbar_T (momenta
 * mom_x[n][3][3], mom_xbar[nbar][3][3] = (pB, pC, pD) per event), form
 * A = I + IV and B = II + III in that order (each part in input order), run the
 * permutation test on (A, B) in the same coordinates, and return the P-even T
 * of (I+II) vs (III+IV) from the same pass. */
et_status et_podd_test(et_ctx *ctx, const void *x, const double *mom_x, int64_t n,
                       const void *xbar, const double *mom_xbar, int64_t nbar,
                       int dim, et_dtype dtype, et_memspace mem, double sigma,
                       int64_t nperm, uint64_t seed, double *T_perm, et_podd_result *out);

/* Eq. 2 (weighted if wx, wxbar are given; both NULL otherwise) for nsig <= ET_MAX_SIGMAS values of
 * sigma from ONE pass over the pairs: the sigma scan of Sect. 2.2 (Fig. 2) evaluates the
 * same samples at several sigma, and d_ij does not depend on sigma.  out[nsig] (host) receives one
 * et_result per sigma, each within the tolerance of the corresponding et_T / et_T_weighted call.
 * ET_ERR_SIGMA if a sigma is not finite and > 0 or two of them differ by more than a factor 1e6. */
#define ET_MAX_SIGMAS 4
et_status et_T_sigmas(et_ctx *ctx, const void *x, const double *wx, int64_t n,
                      const void *xbar, const double *wxbar, int64_t nbar,
                      int dim, et_dtype dtype, et_memspace mem,
                      const double *sigmas, int nsig, et_result *out);

/* Result of et_T_bkg: Eq. 3 and its three normalised brackets, T = T_xx + T_bb - T_xb. */
typedef struct {
    double T, T_xx, T_bb, T_xb;
    double S[10];       /* raw psi sums over unordered pairs (i < j within a sample, all pairs across), in the
                           order XX, XBx, XXbar, XBxbar, BxBx, BxXbar, BxBxbar, XbarXbar, XbarBxbar, BxbarBxbar */
    double w, wbar;     /* signal events in the main samples: n - b, nbar - bbar                             */
    int64_t n_pairs;    /* unordered pairs evaluated                                                         */
} et_bkg_result;

/* Background-subtracted T of Eq. 3 (readings R8, R9): main
 * samples x[n][dim], xbar[nbar][dim], background samples bx[bs][dim],
 * bxbar[bsbar][dim] (all the same dtype and memory space), b and bbar the
 * numbers of background events IN THE MAIN samples (real, >= 0).  All ten
 * sample-pair sums come from one all-pairs pass over the four samples.
 * ET_ERR_INVALID if a sample has < 2 events or b, bbar are negative or not
 * finite; ET_ERR_DEGENERATE if n - b <= 1 or nbar - bbar <= 1.  With
 * b = bbar = 0 the result is Eq. 2 of (x, xbar). */
et_status et_T_bkg(et_ctx *ctx, const void *x, int64_t n, const void *xbar, int64_t nbar,
                   const void *bx, int64_t bs, const void *bxbar, int64_t bsbar,
                   double b, double bbar, int dim, et_dtype dtype, et_memspace mem,
                   double sigma, et_bkg_result *out);

/* Permutation test with Eq. 3 as the statistic (the permutation method is used "using the same
 * method to remove background from the randomly permuted samples"; reading R18 of DESIGN.md).  Permutation p
 * reassigns the pooled main events to main samples of sizes (n, nbar) with the labels of reading R4 drawn from
 * `seed`, and the pooled background-sample events to samples of sizes (bs, bsbar) with the labels drawn from
 * seed ^ 0x9E3779B97F4A7C15; a random flavour gives both main samples the same purity, so the permuted samples
 * are evaluated with b' = (b + bbar) n / (n + nbar) and bbar' = (b + bbar) nbar / (n + nbar).  One four-class
 * all-pairs pass per permutation (the paper's cost model; meant for background studies of modest size).
 * T_perm[nperm] is host memory; ET_OPT_PERM_OFFSET applies. */
typedef struct {
    et_bkg_result observed;
    double p_value;                  /* count_gt / nperm                                              */
    int64_t count_gt, n_near, nperm; /* as et_perm_result                                             */
} et_bkg_perm_result;

et_status et_bkg_permutation_test(et_ctx *ctx, const void *x, int64_t n, const void *xbar, int64_t nbar,
                                  const void *bx, int64_t bs, const void *bxbar, int64_t bsbar,
                                  double b, double bbar, int dim, et_dtype dtype, et_memspace mem,
                                  double sigma, int64_t nperm, uint64_t seed,
                                  double *T_perm, et_bkg_perm_result *out);

/* GEV fit of the permutation T values ("the permutation T distribution can be fitted with a
 * generalised-extreme-value (GEV) function ... The p-value from the fitted T distribution can be calculated as
 * the fraction of the integral of the function above the observed T value"; its uncertainty "by
 * randomly resampling the fit parameters within their uncertainties, taking into account their correlations").
 * F(x) = exp(-t^(-1/xi)), t = 1 + xi (x - mu) / sigma  (xi -> 0: Gumbel; xi > 0 is the heavy upper tail). */
typedef struct {
    double mu, sigma, xi;     /* maximum-likelihood location, scale, shape                                    */
    double cov[9];            /* covariance of (mu, sigma, xi), row-major: inverse observed information; NaN if
                                 it is not positive definite                                                   */
    double nll;               /* negative log-likelihood at the optimum                                        */
    double p_value;           /* 1 - F(T_obs) of the fitted function                                           */
    double p_lo, p_med, p_hi; /* 15.9 %, 50 %, 84.1 % quantiles of the p-values of the resampled parameter sets
                                 (NaN if nresample == 0 or no covariance)                                      */
    int64_t n_used;           /* finite T_perm values that entered the fit                                     */
    int64_t converged;        /* 1: simplex restarts agree and the covariance is positive definite             */
    int64_t n_resampled;      /* parameter sets with sigma > 0 that entered the quantiles                      */
} et_gev_result;

/* Host-only post-processing, O(nperm): all pointers are host memory, no context and no GPU work.  T_perm[nperm]
 * as returned by et_permutation_test / et_podd_test (non-finite entries are skipped; >= 10 finite values with
 * non-zero spread are required, else ET_ERR_DEGENERATE).  z[nresample][3] are the caller's standard normal
 * draws for the parameter resampling theta = theta_hat + L z, cov = L L^T (nresample may be 0, z NULL): the
 * library draws no random numbers here, so the result is a pure function of its inputs. */
et_status et_gev_pvalue(const double *T_perm, int64_t nperm, double T_obs,
                        const double *z, int64_t nresample, et_gev_result *out);

/* Binned S_CP chi^2 of Sect. 2.1 (Eq. 1): the paper's comparison method.
 *   S_CP^i = (N^i(X) - alpha N^i(Xbar)) / sqrt(N^i(X) + alpha^2 N^i(Xbar)),  alpha = N_tot(X) / N_tot(Xbar),
 *   chi^2 = sum_i (S_CP^i)^2, ndf = bins - 1, p = upper tail of chi^2(ndf).
 * The paper leaves the binning to the analyst; readings R19-R21 of DESIGN.md: a uniform rectangular
 * grid, axis k has nbins[k] equal bins over [lo[k], hi[k]] (lo, hi, nbins: HOST arrays [dim], lo < hi, nbins >= 1,
 * product <= 2^24); bin = floor(((x - lo) / (hi - lo)) nbins) in fp64 in this order, x == hi in the last bin, flat
 * index with axis 0 slowest; events outside the box (or not finite) are left out and counted in n_outside; N_tot are
 * the yields inside the grid; a bin empty in both samples is not a bin (S = 0, not counted in ndf).
 * S, Nx, Nxbar: optional HOST outputs [product of nbins] (NULL to skip).  ET_ERR_DEGENERATE when a sample has no
 * event inside the grid or fewer than two bins have entries.  Here n, nbar >= 1 suffice and sigma plays no role. */
typedef struct {
    double chi2;
    int64_t ndf;           /* bins with entries - 1                                              */
    double p_value;        /* Q(ndf / 2, chi2 / 2)                                               */
    double alpha;
    int64_t n_in_x, n_in_xbar, n_outside;
    int64_t bins_used, bins_total;
} et_scp_result;

et_status et_scp(et_ctx *ctx, const void *x, int64_t n, const void *xbar, int64_t nbar,
                 int dim, et_dtype dtype, et_memspace mem,
                 const double *lo, const double *hi, const int32_t *nbins,
                 double *S, int64_t *Nx, int64_t *Nxbar, et_scp_result *out);

/* Test hook: the permutation labels of reading R4, bit-packed,
 * mask[i * ceil(nperm/32) + (p >> 5)] bit (p & 31) = 1 iff pooled event i is in
 * sample X of permutation p.  `mask` lives in `mem`. */
et_status et_perm_labels(et_ctx *ctx, int64_t N, int64_t n, int64_t nperm, uint64_t seed,
                         et_memspace mem, uint32_t *mask);

/* Test hook: per-row class sums for the listed pooled rows (host int64),
 *   r_x[k] = sum_{j in X, j != i} w_j psi_ij,  r_xbar[k] = sum_{j in Xbar, j != i} w_j psi_ij
 * (w = 1 when wx == wxbar == NULL).  r_x, r_xbar are host arrays [nrows]. */
et_status et_row_sums(et_ctx *ctx, const void *x, const double *wx, int64_t n,
                      const void *xbar, const double *wxbar, int64_t nbar,
                      int dim, et_dtype dtype, et_memspace mem, double sigma,
                      const int64_t *rows, int64_t nrows, double *r_x, double *r_xbar);

/* ---- The entry point that allocates nothing (csrc/et_static.cu) --------------------------------------
 * For callers that cannot call cudaMalloc: code under CUDA graph capture, tight serving loops, harnesses
 * that forbid allocation.  et_T_static evaluates Eq. 2 like et_T, but all of its scratch (the
 * bounding box, the pooled fp32 records, the per-CTA partial sums) is ONE file-scope static __device__
 * array of ET_STATIC_SCRATCH_BYTES that every GPU loading libet.so holds until exit.  It needs no context.
 *
 *   et_static_setup(device): once per device, BEFORE any capture: resolves the device address of the array
 *     (cudaGetSymbolAddress with that device current; the caller's current device is restored).  Idempotent.
 *   et_T_static(device, cuda_stream, x, n, xbar, nbar, dim, dtype, sigma, out_device):
 *     x[n][dim], xbar[nbar][dim] are DEVICE pointers on `device`, complete as seen from `cuda_stream` (NULL =
 *     the legacy default stream); out_device is a DEVICE et_result owned by the caller (8-byte aligned).  The call
 *     enqueues five kernels on the stream and returns WITHOUT synchronising: it calls no cudaMalloc, cudaFree,
 *     cudaMallocHost, creates no stream or event, and copies nothing to the host; the caller synchronises the
 *     stream (or launches the captured graph) before reading *out_device.  Makes `device` current.
 *     Limit: 65536 + npad * 4 * ceil((dim + 1) / 4) * 4 bytes <= ET_STATIC_SCRATCH_BYTES, npad = n and nbar
 *     each rounded up to 1024 -- about 5.2e5 pooled events at dim <= 3, 2.6e5 at dim 4..7, 1.7e5 at dim 8
 *     (BASELINE configs 0, 1 and 3 fit, configs 2 and 4 do not); a larger call returns ET_ERR_INVALID and
 *     enqueues nothing.  Other errors: ET_ERR_INVALID (null pointer, n < 2, nbar < 2, dim, dtype, set-up
 *     missing), ET_ERR_SIGMA, ET_ERR_CUDA (a launch failed).  Non-finite coordinates cannot be reported
 *     without a synchronisation: T, the three terms and the three sums of *out_device are then NaN.
 *     Every call shares the array and finds the last call's contents in it; the kernels reset or overwrite
 *     what they use.  Calls that overlap on the GPU (two streams, two host threads, two graphs in flight) RACE
 *     on the array: the caller serialises them.  Arithmetic: that of et_T's difference form (fp32 per pair,
 *     fp64 sums, fixed order): the result agrees with et_T to rounding order.
 *   et_static_last_error(): message of the calling thread's last failed et_static_setup / et_T_static. */
#define ET_STATIC_SCRATCH_BYTES (8u << 20)
et_status et_static_setup(int device);
et_status et_T_static(int device, void *cuda_stream, const void *x, int64_t n, const void *xbar, int64_t nbar,
                      int dim, et_dtype dtype, double sigma, et_result *out_device);
const char *et_static_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* ET_H_ */
