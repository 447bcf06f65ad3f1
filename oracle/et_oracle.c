/*
 * et_oracle.c -- TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, double-precision CPU statement of what the energy-test hot path
 * computes, written from the paper (arXiv:1612.04705, /root/reference/PAPER.md)
 * and from the readings listed in DESIGN.md.  It is the oracle the CUDA path is
 * compared against.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may load it.  It shares no code, header,
 * table or helper with paper_1612_04705_b200/csrc/ and neither includes the
 * other.
 *
 * Every function is the definition written out as loops over pairs: no
 * blocking, no fusion, no Q/R/S identity, no reuse of psi between
 * permutations.  `#pragma omp parallel for reduction` on the outer event loop
 * is the only concession (fp64 sums, so the order change is ~1e-16 relative).
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): closed forms P1-P4, the
 * symmetries P5, the exhaustive-permutation zero mean P6, brute-force p-values
 * P8, the Random123 Philox4x32-10 known answers P9, label counts P10, the
 * duplicated-event identity for integer weights P11, Eq. 3 as a special case
 * P12, the unit-cube expectation P13, the triple-product symmetries P14.
 * Parity unpinned: the value of T on large samples (the paper prints no T or
 * p for any reproducible input) -- pinned only oracle-vs-GPU.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    double T, T_xx, T_bb, T_xb; /* Eq. 2 and its three normalised terms (T = T_xx + T_bb - T_xb) */
    double S_xx, S_bb, S_xb;    /* raw psi sums: i<j within X, i<j within Xbar, all (i,j) across */
    double W, Wbar;             /* n, nbar (unweighted) or the weight sums                      */
    int64_t n_pairs;            /* n(n-1)/2 + nbar(nbar-1)/2 + n*nbar                             */
} oracle_result;

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* psi_ij = exp(-d_ij^2 / (2 sigma^2)), d_ij the Euclidean length of the
 * coordinate displacement vector.  PAPER.md:71 (Sect. 2.2), :119 (Sect. 4.1). */
double oracle_psi(const double *a, const double *b, int dim, double sigma)
{
    double d2 = 0.0;
    for (int k = 0; k < dim; ++k) {
        double d = a[k] - b[k];
        d2 += d * d;
    }
    return exp(-d2 / (2.0 * sigma * sigma));
}

/* Eq. 2 with per-event weights (reading R7):
 *   T = sum_{i<j in X} w_i w_j psi / (W (W-1)) + sum_{i<j in Xbar} ... / (Wbar (Wbar-1))
 *       - sum_{i in X, j in Xbar} w_i w_j psi / (W Wbar),     W = sum_X w, Wbar = sum_Xbar w.
 * wx == NULL / wxbar == NULL means all weights 1, which is Eq. 2 as printed
 * (within terms are half-means, reading R1).
 * Returns 0, -1 invalid arguments, -2 bad sigma, -4 degenerate normalisation. */
int oracle_T_weighted(const double *x, const double *wx, int64_t n,
                      const double *xbar, const double *wxbar, int64_t nbar,
                      int dim, double sigma, oracle_result *out)
{
    if (!x || !xbar || !out || n < 2 || nbar < 2 || dim < 1) return -1;
    if (!(sigma > 0.0) || !isfinite(sigma)) return -2;

    double W = 0.0, Wbar = 0.0;
    for (int64_t i = 0; i < n; ++i) W += wx ? wx[i] : 1.0;
    for (int64_t i = 0; i < nbar; ++i) Wbar += wxbar ? wxbar[i] : 1.0;
    if (!(W > 1.0) || !(Wbar > 1.0)) return -4;

    double S_xx = 0.0, S_bb = 0.0, S_xb = 0.0;

#pragma omp parallel for schedule(dynamic, 16) reduction(+ : S_xx)
    for (int64_t i = 0; i < n; ++i) {
        double wi = wx ? wx[i] : 1.0, s = 0.0;
        for (int64_t j = i + 1; j < n; ++j)
            s += (wx ? wx[j] : 1.0) * oracle_psi(x + i * dim, x + j * dim, dim, sigma);
        S_xx += wi * s;
    }
#pragma omp parallel for schedule(dynamic, 16) reduction(+ : S_bb)
    for (int64_t i = 0; i < nbar; ++i) {
        double wi = wxbar ? wxbar[i] : 1.0, s = 0.0;
        for (int64_t j = i + 1; j < nbar; ++j)
            s += (wxbar ? wxbar[j] : 1.0) * oracle_psi(xbar + i * dim, xbar + j * dim, dim, sigma);
        S_bb += wi * s;
    }
#pragma omp parallel for schedule(dynamic, 16) reduction(+ : S_xb)
    for (int64_t i = 0; i < n; ++i) {
        double wi = wx ? wx[i] : 1.0, s = 0.0;
        for (int64_t j = 0; j < nbar; ++j)
            s += (wxbar ? wxbar[j] : 1.0) * oracle_psi(x + i * dim, xbar + j * dim, dim, sigma);
        S_xb += wi * s;
    }

    out->S_xx = S_xx;
    out->S_bb = S_bb;
    out->S_xb = S_xb;
    out->W = W;
    out->Wbar = Wbar;
    out->T_xx = S_xx / (W * (W - 1.0));
    out->T_bb = S_bb / (Wbar * (Wbar - 1.0));
    out->T_xb = S_xb / (W * Wbar);
    out->T = out->T_xx + out->T_bb - out->T_xb;
    out->n_pairs = n * (n - 1) / 2 + nbar * (nbar - 1) / 2 + n * nbar;
    return 0;
}

/* Eq. 2, unweighted. */
int oracle_T(const double *x, int64_t n, const double *xbar, int64_t nbar,
             int dim, double sigma, oracle_result *out)
{
    return oracle_T_weighted(x, NULL, n, xbar, NULL, nbar, dim, sigma, out);
}

/* Per-row class sums, for sampled parity at sizes where a full T is too slow
 * (SURVEY.md 8(d)).  Pooled index convention: X events 0..n-1, Xbar events
 * n..n+nbar-1.  For each listed pooled row i:
 *   r_x[k]    = sum_{j in X,    j != i} w_j psi_ij
 *   r_xbar[k] = sum_{j in Xbar, j != i} w_j psi_ij        (w = 1 when NULL). */
int oracle_row_sums(const double *x, const double *wx, int64_t n,
                    const double *xbar, const double *wxbar, int64_t nbar,
                    int dim, double sigma, const int64_t *rows, int64_t nrows,
                    double *r_x, double *r_xbar)
{
    if (!x || !xbar || !rows || !r_x || !r_xbar || n < 1 || nbar < 1 || dim < 1) return -1;
    if (!(sigma > 0.0) || !isfinite(sigma)) return -2;
    int bad = 0;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t k = 0; k < nrows; ++k) {
        int64_t i = rows[k];
        if (i < 0 || i >= n + nbar) {
#pragma omp atomic write
            bad = 1;
            continue;
        }
        const double *pi = i < n ? x + i * dim : xbar + (i - n) * dim;
        double sx = 0.0, sb = 0.0;
        for (int64_t j = 0; j < n; ++j)
            if (j != i) sx += (wx ? wx[j] : 1.0) * oracle_psi(pi, x + j * dim, dim, sigma);
        for (int64_t j = 0; j < nbar; ++j)
            if (j + n != i) sb += (wxbar ? wxbar[j] : 1.0) * oracle_psi(pi, xbar + j * dim, dim, sigma);
        r_x[k] = sx;
        r_xbar[k] = sb;
    }
    return bad ? -1 : 0;
}

/* Philox4x32-10 (Salmon et al., SC'11; reading R4 fixes it as the label
 * generator).  Ten rounds of
 *   (hi0,lo0) = 0xD2511F53 * c0,  (hi1,lo1) = 0xCD9E8D57 * c2,
 *   c <- (hi1 ^ c1 ^ k0, lo1, hi0 ^ c3 ^ k1, lo0),
 * the key bumped by (0x9E3779B9, 0xBB67AE85) between rounds. */
void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

static int cmp_u64(const void *a, const void *b)
{
    uint64_t x = *(const uint64_t *)a, y = *(const uint64_t *)b;
    return (x > y) - (x < y);
}

/* Reading R4 ("randomly assigning events to either of the
 * samples", sizes kept): for permutation p and pooled event i
 *   out   = philox(ctr = (i & 0xffffffff, i >> 32, p >> 2, 0), key = (seed lo, seed hi))
 *   key32 = out[p & 3],   K = (key32 << 32) | (uint32) i
 * and event i is in sample X of permutation p iff K is among the n smallest
 * composites of that permutation.  a[(p - p_begin) * N + i] = 1 for X, 0 for Xbar. */
int oracle_labels_range(int64_t N, int64_t n, int64_t p_begin, int64_t p_count,
                        uint64_t seed, uint8_t *a)
{
    if (!a || N < 1 || n < 0 || n > N || p_begin < 0 || p_count < 0 || N > 0xffffffffLL) return -1;
    int fail = 0;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t q = 0; q < p_count; ++q) {
        int64_t p = p_begin + q;
        uint64_t *K = (uint64_t *)malloc(sizeof(uint64_t) * (size_t)N);
        uint64_t *sorted = (uint64_t *)malloc(sizeof(uint64_t) * (size_t)N);
        if (!K || !sorted) {
#pragma omp atomic write
            fail = 1;
            free(K);
            free(sorted);
            continue;
        }
        uint32_t key[2] = { (uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32) };
        for (int64_t i = 0; i < N; ++i) {
            uint32_t ctr[4] = { (uint32_t)((uint64_t)i & 0xffffffffu), (uint32_t)((uint64_t)i >> 32),
                                (uint32_t)((uint64_t)p >> 2), 0u };
            uint32_t out[4];
            oracle_philox4x32_10(ctr, key, out);
            K[i] = ((uint64_t)out[p & 3] << 32) | (uint32_t)i;
        }
        memcpy(sorted, K, sizeof(uint64_t) * (size_t)N);
        qsort(sorted, (size_t)N, sizeof(uint64_t), cmp_u64);
        uint8_t *row = a + (size_t)q * (size_t)N;
        if (n == 0) {
            memset(row, 0, (size_t)N);
        } else {
            uint64_t thr = sorted[n - 1]; /* the n-th smallest; composites are distinct */
            for (int64_t i = 0; i < N; ++i) row[i] = K[i] <= thr;
        }
        free(K);
        free(sorted);
    }
    return fail ? -5 : 0;
}

/* Bit-packed form: mask[i * nwords + (p >> 5)] bit (p & 31), nwords = ceil(nperm / 32). */
int oracle_labels(int64_t N, int64_t n, int64_t nperm, uint64_t seed, uint32_t *mask)
{
    if (!mask || nperm < 1) return -1;
    int64_t nwords = (nperm + 31) / 32;
    memset(mask, 0, sizeof(uint32_t) * (size_t)N * (size_t)nwords);
    uint8_t *a = (uint8_t *)malloc((size_t)N);
    if (!a) return -5;
    for (int64_t p = 0; p < nperm; ++p) {
        int rc = oracle_labels_range(N, n, p, 1, seed, a);
        if (rc) { free(a); return rc; }
        for (int64_t i = 0; i < N; ++i)
            if (a[i]) mask[i * nwords + (p >> 5)] |= 1u << (p & 31);
    }
    free(a);
    return 0;
}

typedef struct {
    oracle_result observed;
    double p_value;
    int64_t count_gt, nperm;
} oracle_perm_result;

/* Permutation test: pool the events, reassign them to two samples
 * of the original sizes (labels as above), evaluate Eq. 2 (or its weighted form,
 * the weights travelling with their events, reading R10) FROM SCRATCH on each
 * split; p = #{T_p > T_obs} / nperm (strict, reading R3).  A degenerate split
 * (W_p <= 1 or Wbar_p <= 1) gives T_p = NaN and is not counted. */
int oracle_perm_test(const double *x, const double *wx, int64_t n,
                     const double *xbar, const double *wxbar, int64_t nbar,
                     int dim, double sigma, int64_t nperm, uint64_t seed,
                     double *T_perm, oracle_perm_result *out)
{
    if (!T_perm || !out || nperm < 1) return -1;
    if ((wx == NULL) != (wxbar == NULL)) return -1;
    int rc = oracle_T_weighted(x, wx, n, xbar, wxbar, nbar, dim, sigma, &out->observed);
    if (rc) return rc;

    int64_t N = n + nbar;
    size_t row = sizeof(double) * (size_t)dim;
    uint8_t *a = (uint8_t *)malloc((size_t)N);
    double *px = (double *)malloc(row * (size_t)n), *pb = (double *)malloc(row * (size_t)nbar);
    double *pwx = wx ? (double *)malloc(sizeof(double) * (size_t)n) : NULL;
    double *pwb = wx ? (double *)malloc(sizeof(double) * (size_t)nbar) : NULL;
    if (!a || !px || !pb || (wx && (!pwx || !pwb))) { free(a); free(px); free(pb); free(pwx); free(pwb); return -5; }

    int64_t count = 0;
    for (int64_t p = 0; p < nperm; ++p) {
        rc = oracle_labels_range(N, n, p, 1, seed, a);
        if (rc) break;
        int64_t kx = 0, kb = 0;
        for (int64_t i = 0; i < N; ++i) {
            const double *src = i < n ? x + i * dim : xbar + (i - n) * dim;
            double w = wx ? (i < n ? wx[i] : wxbar[i - n]) : 1.0;
            if (a[i]) { memcpy(px + kx * dim, src, row); if (wx) pwx[kx] = w; ++kx; }
            else      { memcpy(pb + kb * dim, src, row); if (wx) pwb[kb] = w; ++kb; }
        }
        oracle_result r;
        int rp = oracle_T_weighted(px, pwx, kx, pb, pwb, kb, dim, sigma, &r);
        if (rp == -4) { T_perm[p] = NAN; continue; }
        if (rp) { rc = rp; break; }
        T_perm[p] = r.T;
        if (r.T > out->observed.T) ++count;
    }
    free(a); free(px); free(pb); free(pwx); free(pwb);
    if (rc) return rc;
    out->count_gt = count;
    out->nperm = nperm;
    out->p_value = (double)count / (double)nperm;
    return 0;
}

/* Sect. 5 split (Eq. 4; reading R11).  Triple product
 * C = pB . (pC x pD) of three final-state momenta in the mother rest frame.
 * For a D (is_conjugate = 0) the event is "positive" (class I) iff C_T > 0;
 * for a Dbar (is_conjugate = 1) the momenta supplied are those of the
 * C-conjugate particles, C = Cbar_T, and the event is positive (class III) iff
 * -Cbar_T > 0.  C exactly 0 goes to the negative class (II / IV). */
int oracle_podd_split(const double *pB, const double *pC, const double *pD, int64_t n,
                      int is_conjugate, uint8_t *positive, int64_t *n_positive)
{
    if (!pB || !pC || !pD || !positive || n < 0) return -1;
    int64_t cnt = 0;
    for (int64_t i = 0; i < n; ++i) {
        const double *b = pB + 3 * i, *c = pC + 3 * i, *d = pD + 3 * i;
        double cx = c[1] * d[2] - c[2] * d[1];
        double cy = c[2] * d[0] - c[0] * d[2];
        double cz = c[0] * d[1] - c[1] * d[0];
        double C = b[0] * cx + b[1] * cy + b[2] * cz;
        double v = is_conjugate ? -C : C;
        positive[i] = v > 0.0;
        cnt += positive[i];
    }
    if (n_positive) *n_positive = cnt;
    return 0;
}

/* Eq. 3 (readings R8, R9): background-subtracted T from the
 * main samples X (n events), Xbar (nbar) and the background samples Bx (bs
 * events), Bxbar (bsbar), with b, bbar the numbers of background events in the
 * main samples and w = n - b, wbar = nbar - bbar the numbers of signal events.
 * Sums over i != j (both orders) with the factor 1/2, exactly as printed. */
static double sum_ne(const double *a, int64_t na, int dim, double sigma)
{
    double s = 0.0;
#pragma omp parallel for schedule(dynamic, 16) reduction(+ : s)
    for (int64_t i = 0; i < na; ++i)
        for (int64_t j = 0; j < na; ++j)
            if (j != i) s += oracle_psi(a + i * dim, a + j * dim, dim, sigma);
    return s;
}
static double sum_cross(const double *a, int64_t na, const double *b, int64_t nb, int dim, double sigma)
{
    double s = 0.0;
#pragma omp parallel for schedule(dynamic, 16) reduction(+ : s)
    for (int64_t i = 0; i < na; ++i)
        for (int64_t j = 0; j < nb; ++j) s += oracle_psi(a + i * dim, b + j * dim, dim, sigma);
    return s;
}
int oracle_T_bkg(const double *x, int64_t n, const double *xbar, int64_t nbar,
                 const double *bx, int64_t bs, const double *bxbar, int64_t bsbar,
                 double b, double bbar, int dim, double sigma, double *T_out)
{
    if (!x || !xbar || !bx || !bxbar || !T_out || n < 2 || nbar < 2 || bs < 2 || bsbar < 2 || dim < 1) return -1;
    if (!(sigma > 0.0) || !isfinite(sigma)) return -2;
    double w = (double)n - b, wbar = (double)nbar - bbar;
    if (!(w > 1.0) || !(wbar > 1.0)) return -4;
    double dbs = (double)bs, dbsb = (double)bsbar;
    double t1 = sum_ne(x, n, dim, sigma)
              - 2.0 * b / dbs * sum_cross(x, n, bx, bs, dim, sigma)
              + b * (b + 1.0) / (dbs * (dbs - 1.0)) * sum_ne(bx, bs, dim, sigma);
    double t2 = sum_ne(xbar, nbar, dim, sigma)
              - 2.0 * bbar / dbsb * sum_cross(xbar, nbar, bxbar, bsbar, dim, sigma)
              + bbar * (bbar + 1.0) / (dbsb * (dbsb - 1.0)) * sum_ne(bxbar, bsbar, dim, sigma);
    double t3 = sum_cross(x, n, xbar, nbar, dim, sigma)
              - bbar / dbsb * sum_cross(x, n, bxbar, bsbar, dim, sigma)
              - b / dbs * sum_cross(xbar, nbar, bx, bs, dim, sigma)
              + b * bbar / (dbs * dbsb) * sum_cross(bx, bs, bxbar, bsbar, dim, sigma);
    *T_out = t1 / (2.0 * w * (w - 1.0)) + t2 / (2.0 * wbar * (wbar - 1.0)) - t3 / (w * wbar);
    return 0;
}
