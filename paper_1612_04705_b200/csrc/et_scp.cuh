// et_scp.cuh -- the binned S_CP chi^2 of Sect. 2.1 (Eq. 1 at :29), the paper's comparison method
// (SURVEY 8(f) NEXT-4): one histogram pass per sample and one reduction.  O(N), HBM-bound: 8 dim bytes per event.
//   S_CP^i = (N^i(X) - alpha N^i(Xbar)) / sqrt(N^i(X) + alpha^2 N^i(Xbar)),  alpha = N_tot(X) / N_tot(Xbar),
//   chi^2 = sum_i (S_CP^i)^2,  ndf = bins - 1.
// Readings R19-R21: uniform rectangular grid, bin = floor(((x - lo) / (hi - lo)) nbins) in fp64 in exactly
// this order without contraction (the bin of an event is an integer decision: it must be the one a plain fp64 CPU
// evaluation takes), x == hi in the last bin, events outside the box counted apart; N_tot = yields inside the grid; a
// bin empty in both samples is not a bin.
#pragma once
#include <cmath>

#include "et_device.cuh"

namespace et {
namespace scp {

constexpr int kMaxAxes = 8;
constexpr int kSmemBins = 8192;           // histograms up to this many bins are accumulated in shared memory first
constexpr long long kMaxBins = 1ll << 24;

struct Grid {
    double lo[kMaxAxes], hi[kMaxAxes];
    int nbins[kMaxAxes];
    int dim;
    int total;
};

template <typename TIn>
__device__ __forceinline__ int bin_of(const TIn *__restrict__ p, const Grid &G)
{
    int flat = 0;
    bool inside = true;
#pragma unroll 1
    for (int k = 0; k < G.dim; ++k) {
        const double v = (double)p[k];
        const bool ok = (v >= G.lo[k]) && (v <= G.hi[k]);  // false for NaN
        const double t = __ddiv_rn(__dsub_rn(v, G.lo[k]), __dsub_rn(G.hi[k], G.lo[k]));
        int b = ok ? (int)floor(__dmul_rn(t, (double)G.nbins[k])) : 0;
        b = min(b, G.nbins[k] - 1);
        inside = inside && ok;
        flat = flat * G.nbins[k] + b;
    }
    return inside ? flat : -1;
}

// counts[bin] += 1 for every event of one sample, *outside += events not in the grid.  Integer atomics: the result
// does not depend on their order.
template <typename TIn, bool SMEM>
__global__ void __launch_bounds__(256) k_scp_hist(const TIn *__restrict__ x, long long n, Grid G, unsigned long long *__restrict__ counts,
                                                  unsigned long long *__restrict__ outside)
{
    __shared__ unsigned int h[SMEM ? kSmemBins : 1];
    if (SMEM) {
        for (int b = threadIdx.x; b < G.total; b += blockDim.x) h[b] = 0u;
        __syncthreads();
    }
    unsigned int out = 0;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const int b = bin_of<TIn>(x + i * G.dim, G);
        if (b < 0) ++out;
        else if (SMEM) atomicAdd(&h[b], 1u);
        else atomicAdd(&counts[b], 1ull);
    }
    for (int o = 16; o > 0; o >>= 1) out += __shfl_xor_sync(0xffffffffu, out, o);
    if ((threadIdx.x & 31) == 0 && out) atomicAdd(outside, (unsigned long long)out);
    if (SMEM) {
        __syncthreads();
        for (int b = threadIdx.x; b < G.total; b += blockDim.x)
            if (h[b]) atomicAdd(&counts[b], (unsigned long long)h[b]);
    }
}

struct DevScp {
    double chi2, alpha;
    long long n_in_x, n_in_xbar, bins_used;
};

// One CTA, fixed order: totals, alpha, then Eq. 1 bin by bin.  S may be null.
__global__ void __launch_bounds__(1024) k_scp_stat(const unsigned long long *__restrict__ Nx, const unsigned long long *__restrict__ Nb, int total,
                                                   double *__restrict__ S, DevScp *out)
{
    __shared__ double sd[1024];
    __shared__ unsigned long long sa[1024], sb[1024];
    const int t = threadIdx.x;
    unsigned long long a = 0, b = 0;
    for (int i = t; i < total; i += 1024) { a += Nx[i]; b += Nb[i]; }
    sa[t] = a; sb[t] = b;
    __syncthreads();
    for (int s = 512; s > 0; s >>= 1) {
        if (t < s) { sa[t] += sa[t + s]; sb[t] += sb[t + s]; }
        __syncthreads();
    }
    const unsigned long long ntx = sa[0], ntb = sb[0];
    __syncthreads();
    const double alpha = __ddiv_rn((double)ntx, (double)ntb);
    double c = 0.0;
    unsigned long long used = 0;
    for (int i = t; i < total; i += 1024) {
        const double nx = (double)Nx[i], nb = (double)Nb[i];
        double s = 0.0;
        if (Nx[i] | Nb[i]) {
            ++used;
            const double num = __dsub_rn(nx, __dmul_rn(alpha, nb));
            const double den = sqrt(__dadd_rn(nx, __dmul_rn(__dmul_rn(alpha, alpha), nb)));
            s = __ddiv_rn(num, den);
            c = __dadd_rn(c, __dmul_rn(s, s));
        }
        if (S) S[i] = s;
    }
    sd[t] = c; sa[t] = used;
    __syncthreads();
    for (int s = 512; s > 0; s >>= 1) {
        if (t < s) { sd[t] += sd[t + s]; sa[t] += sa[t + s]; }
        __syncthreads();
    }
    if (t == 0) {
        out->chi2 = sd[0];
        out->alpha = alpha;
        out->n_in_x = (long long)ntx;
        out->n_in_xbar = (long long)ntb;
        out->bins_used = (long long)sa[0];
    }
}

// Upper tail of the chi^2 distribution with ndf degrees of freedom: Q(ndf / 2, chi2 / 2), the regularised upper incomplete
// gamma function, by its power series (x < a + 1) or Lentz's continued fraction (host, O(1)).
inline double chi2_sf(double chi2, long long ndf)
{
    if (!(ndf > 0) || !(chi2 >= 0.0)) return std::nan("");
    const double a = 0.5 * (double)ndf, x = 0.5 * chi2;
    if (x == 0.0) return 1.0;
    const double lg = std::lgamma(a), pre = std::exp(-x + a * std::log(x) - lg);
    if (x < a + 1.0) {
        double term = 1.0 / a, sum = term, ap = a;
        for (int k = 0; k < 100000; ++k) {
            ap += 1.0;
            term *= x / ap;
            sum += term;
            if (std::fabs(term) < std::fabs(sum) * 1e-17) break;
        }
        return 1.0 - pre * sum;
    }
    const double tiny = 1e-300;
    double b = x + 1.0 - a, c = 1.0 / tiny, d = 1.0 / b, h = d;
    for (int k = 1; k < 100000; ++k) {
        const double an = -(double)k * ((double)k - a);
        b += 2.0;
        d = an * d + b;
        if (std::fabs(d) < tiny) d = tiny;
        c = b + an / c;
        if (std::fabs(c) < tiny) c = tiny;
        d = 1.0 / d;
        const double del = d * c;
        h *= del;
        if (std::fabs(del - 1.0) < 1e-16) break;
    }
    return pre * h;
}

}  // namespace scp
}  // namespace et
