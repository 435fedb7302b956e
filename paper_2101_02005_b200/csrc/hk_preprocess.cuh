// hk_preprocess.cuh -- steps a1-a3 of the hot path:
//   line_kernel   : per-line S, Gamma_L, alpha_D, centre bin, extent, sort key   (Eq. 5, 9, 13; L236-239)
//   gather_kernel : permute records into centre-bin order, apply the launch scale
//   range_kernel  : per warp tile, the candidate line range and its far-interior parts (L347)
//   unit_kernel   : per CTA tile, number of (tile, line-chunk) work units
#pragma once
#include "hk_device.cuh"

namespace hk {

struct Params {
    // grid
    double numin, dnu;
    int64_t N;
    // conditions folded into constants (host, fp64)
    double c2_over_T;     // h c / (k_B T)
    double tfac;          // T_ref / T
    double P_atm;
    double beta;          // sqrt(2 k_B T / m) / c     (alpha_D = beta nu0)
    double sfac;          // 1 / (8 pi c m Q)
    double inv4pic;       // 1 / (4 pi c)
    // cut
    double cut;           // cm^-1 (ignored when uncut)
    int uncut;
    // sort keys: key = jc - kmin in [0, ksent), ksent = sentinel for lines that contribute nothing
    int64_t kmin;
    int32_t ksent;
    // tile ranges
    int64_t cb_floor, cb_ceil;  // floor/ceil of cut/dnu (bins)
    double kappa1, kappa2;      // sqrt(Z1) * beta and sqrt(Z2) * beta, slightly inflated
    double numin_bins;          // numin / dnu
    int32_t kb;                 // bins per lane (2, 4, 8)
    int32_t n_ct;               // tiles of 32 kb bins
    int32_t chunk;              // lines per work unit
    int mode;                   // debug: 0 default, 1 everything through the near kernel, 2 far pairs through the mid kernel
};

struct DevStats {
    unsigned long long n_skipped, n_off_grid, n_evals, n_cnt_mid, n_cnt_core;  // cnt_*: evals with |z|^2 below Z1 / Z2
    unsigned long long cmax_bits, cKmax_bits;                                  // max Lorentz amplitude / cK as double bits
    int32_t scale_exp;
    int32_t pad;
    unsigned int unit_counter_far, unit_counter_mid, unit_counter_near, pad2;
    unsigned long long units_far, units_mid, units_near;
    unsigned long long pairs_far, pairs_mid, pairs_near;   // (line, bin) slots per kernel, from the tile ranges
};

__device__ __forceinline__ bool finite6(double a, double b, double c, double d, double e, double f)
{
    return isfinite(a) && isfinite(b) && isfinite(c) && isfinite(d) && isfinite(e) && isfinite(f);
}

struct LineOut {
    bool valid;       // passes the R14 checks
    bool on_grid;     // extent non-empty and centre within 2^30 bins
    double S, gammaL, alphaD;
    int64_t jc, ilo, ihi;
    double pos_f;     // (nu0-numin)/dnu - jc
};

// The fp64 arithmetic of step a1.  Extents use IEEE operations in exactly the order
// SURVEY.md 8(c).4 states (no contraction: explicit _rn intrinsics).
__device__ __forceinline__ LineOut line_math(const Params& p, double nu0, double A, double g, double E,
                                             double gam, double nx)
{
    LineOut o;
    o.valid = finite6(nu0, A, g, E, gam, nx) && nu0 > 0.0 && A >= 0.0;
    o.on_grid = false;
    o.S = o.gammaL = o.alphaD = 0.0;
    o.jc = 0; o.ilo = 0; o.ihi = -1; o.pos_f = 0.0;
    if (!o.valid) return o;
    o.alphaD = p.beta * nu0;                                                   // Eq. 13 (L203)
    o.gammaL = A * p.inv4pic + gam * pow(p.tfac, nx) * p.P_atm;                // Eq. 5 (L91)
    o.S = A * g * p.sfac / (nu0 * nu0) * exp(-p.c2_over_T * E) * (-expm1(-p.c2_over_T * nu0));  // Eq. 9 (L127)
    const double big = 4.0e18;
    double pos = __ddiv_rn(__dsub_rn(nu0, p.numin), p.dnu);
    double c = floor(pos);
    c = fmin(fmax(c, -big), big);
    o.jc = (int64_t)c;
    o.pos_f = pos - c;
    if (!p.uncut) {
        double lo = ceil(__ddiv_rn(__dsub_rn(__dsub_rn(nu0, p.cut), p.numin), p.dnu));
        double hi = floor(__ddiv_rn(__dsub_rn(__dadd_rn(nu0, p.cut), p.numin), p.dnu));
        if (lo < 0.0) lo = 0.0;
        if (hi > (double)(p.N - 1)) hi = (double)(p.N - 1);
        lo = fmin(lo, big);
        hi = fmax(hi, -big);
        o.ilo = (int64_t)lo;
        o.ihi = (int64_t)hi;
    } else {
        o.ilo = 0;
        o.ihi = p.N - 1;
    }
    o.on_grid = (o.ilo <= o.ihi) && (o.jc >= -(1LL << 30)) && (o.jc <= (1LL << 30) - 2);
    return o;
}

// number of integers i in [ilo, ihi] with |i - pos| < T
__device__ __forceinline__ int64_t count_within(double pos, double T, int64_t ilo, int64_t ihi)
{
    if (!(T > 0.0)) return 0;
    double lo = floor(pos - T) + 1.0, hi = ceil(pos + T) - 1.0;
    lo = fmax(lo, (double)ilo);
    hi = fmin(hi, (double)ihi);
    return hi >= lo ? (int64_t)(hi - lo) + 1 : 0;
}

__global__ void __launch_bounds__(256) line_kernel(Params p, const double* __restrict__ nu0,
                                                   const double* __restrict__ A, const double* __restrict__ g,
                                                   const double* __restrict__ E, const double* __restrict__ gam,
                                                   const double* __restrict__ nx, int64_t n, RecU* __restrict__ rec,
                                                   int32_t* __restrict__ key, int32_t* __restrict__ idx,
                                                   DevStats* __restrict__ st)
{
    unsigned long long skipped = 0, off = 0, evals = 0, cmid = 0, ccore = 0, cmaxb = 0, cKmaxb = 0;
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        LineOut o = line_math(p, nu0[i], A[i], g[i], E[i], gam[i], nx[i]);
        RecU r;
        int32_t k = p.ksent;
        r.jc = 0; r.f = 0.f; r.G2 = 0.f; r.a2 = 0.f; r.ilo = 0; r.ihi = -1; r.cK = 0.0;
        if (!o.valid) {
            ++skipped;
        } else if (!o.on_grid) {
            ++off;
            r.jc = (int32_t)max(min(o.jc, (int64_t)INT32_MAX), (int64_t)INT32_MIN);
        } else {
            double Gb = o.gammaL / p.dnu, ab = o.alphaD / p.dnu;
            r.jc = (int32_t)o.jc;
            r.f = fminf((float)o.pos_f, 0.99999994f);
            r.G2 = (float)(Gb * Gb);
            r.a2 = (float)(ab * ab);
            r.ilo = (int32_t)o.ilo;
            r.ihi = (int32_t)o.ihi;
            r.cK = o.S / (o.alphaD * 1.772453850905516027298);          // S/(alpha_D sqrt(pi))
            double cl = o.S * Gb / (kPi * p.dnu);                       // Lorentz amplitude in bin units
            k = (int32_t)(o.jc - p.kmin);
            cmaxb = max(cmaxb, (unsigned long long)__double_as_longlong(cl));
            cKmaxb = max(cKmaxb, (unsigned long long)__double_as_longlong(r.cK));
            evals += (unsigned long long)(o.ihi - o.ilo + 1);
            double pos = (double)o.jc + o.pos_f;
            double t1 = (double)HK_Z1 * ab * ab - Gb * Gb, t2 = (double)HK_Z2 * ab * ab - Gb * Gb;
            cmid += (unsigned long long)count_within(pos, t1 > 0 ? sqrt(t1) : 0.0, o.ilo, o.ihi);
            ccore += (unsigned long long)count_within(pos, t2 > 0 ? sqrt(t2) : 0.0, o.ilo, o.ihi);
        }
        rec[i] = r;
        key[i] = k;
        idx[i] = (int32_t)i;
    }
    // block reduction of the counters
    __shared__ unsigned long long sh[7][8];
    unsigned long long v[7] = {skipped, off, evals, cmid, ccore, cmaxb, cKmaxb};
#pragma unroll
    for (int q = 0; q < 7; ++q) {
        unsigned long long x = v[q];
        for (int o = 16; o > 0; o >>= 1) {
            unsigned long long y = __shfl_xor_sync(0xffffffffu, x, o);
            x = (q < 5) ? x + y : max(x, y);
        }
        if ((threadIdx.x & 31) == 0) sh[q][threadIdx.x >> 5] = x;
    }
    __syncthreads();
    if (threadIdx.x < 7) {
        int q = threadIdx.x;
        unsigned long long x = sh[q][0];
        for (int w = 1; w < 8; ++w) x = (q < 5) ? x + sh[q][w] : max(x, sh[q][w]);
        unsigned long long* dst = q == 0 ? &st->n_skipped : q == 1 ? &st->n_off_grid : q == 2 ? &st->n_evals
                                : q == 3 ? &st->n_cnt_mid : q == 4 ? &st->n_cnt_core : q == 5 ? &st->cmax_bits
                                : &st->cKmax_bits;
        if (q < 5) { if (x) atomicAdd(dst, x); }
        else atomicMax(dst, x);
    }
}

// One thread: power-of-two launch scale from the maxima (max Lorentz amplitude -> 2^40,
// and cK kept below 2^100), DESIGN.md section 4 "dynamic range".
__global__ void scale_kernel(DevStats* st)
{
    double cmax = __longlong_as_double((long long)st->cmax_bits);
    double cKmax = __longlong_as_double((long long)st->cKmax_bits);
    int e = 0;
    if (cmax > 0.0 && isfinite(cmax)) e = 40 - ilogb(cmax);
    if (cKmax > 0.0 && isfinite(cKmax)) e = min(e, 100 - ilogb(cKmax));
    if (!(cmax > 0.0) && cKmax > 0.0 && isfinite(cKmax)) e = 60 - ilogb(cKmax);
    e = max(-900, min(900, e));
    st->scale_exp = e;
}

__global__ void __launch_bounds__(256) gather_kernel(const RecU* __restrict__ rec, const int32_t* __restrict__ idx_sorted,
                                                     int64_t n, const DevStats* __restrict__ st,
                                                     float4* __restrict__ recA, float4* __restrict__ recB)
{
    const int e = st->scale_exp;
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const RecU r = rec[idx_sorted[i]];
        float cK = (float)scalbn(r.cK, e);
        // c = cK * G a / sqrt(pi)  (Lorentz amplitude S Gamma_L/(pi dnu^2) in bin units)
        float c = cK * sqrtf(r.G2 * r.a2) * 0.564189583547756f;
        recA[i] = make_float4(__int_as_float(r.jc), r.f, r.G2, c);
        recB[i] = make_float4(r.a2, __int_as_float(r.ilo), __int_as_float(r.ihi), cK);
    }
}

// first index with key >= v in the sorted key array
__device__ __forceinline__ int32_t lower_bound_key(const int32_t* __restrict__ keys, int32_t n, int64_t v)
{
    int32_t lo = 0, hi = n;
    while (lo < hi) {
        int32_t mid = lo + ((hi - lo) >> 1);
        if ((int64_t)keys[mid] < v) lo = mid + 1; else hi = mid;
    }
    return lo;
}

// Per tile [w0, w1): candidate lines and their split into edge / far / mid / centre ranges.
// A line is "interior" for the tile when every bin of the tile lies inside its extent and at
// |t| >= max(16 KB, sqrt(Z) a): then |z|^2 >= Z for every (line, bin) pair (Z = Z1: far, Z = Z2: mid)
// and the interior kernels may run mask-free.  alpha_D = beta nu0 is a function of the centre, so the
// condition is a bound on the centre bin alone; all bounds are conservative.
__device__ __forceinline__ int64_t left_bound(double w0, double kap, double numin_bins)
{
    // pos + 1 <= (w0 - kap numin_bins) / (1 + kap)   =>   w0 - pos >= kap (numin_bins + pos)
    return (int64_t)floor((w0 - kap * (numin_bins + 1.0)) / (1.0 + kap)) - 3;
}
__device__ __forceinline__ int64_t right_bound(double w1m1, double kap, double numin_bins)
{
    // pos >= (w1 - 1 + kap numin_bins) / (1 - kap)   =>   pos - (w1 - 1) >= kap (numin_bins + pos)
    if (!(kap < 0.9)) return INT64_MAX / 2;
    return (int64_t)ceil((w1m1 + kap * (numin_bins + 1.0)) / (1.0 - kap)) + 3;
}

__global__ void __launch_bounds__(256) range_kernel(Params p, const int32_t* __restrict__ keys, int32_t n,
                                                    TileRange* __restrict__ tr, DevStats* __restrict__ st)
{
    int wt = blockIdx.x * blockDim.x + threadIdx.x;
    if (wt >= p.n_ct) return;
    const int wb = 32 * p.kb;
    const int64_t mind = (int64_t)kMinDistPerKB * p.kb;
    const int64_t w0 = (int64_t)wt * wb;
    const int64_t w1 = min(p.N, w0 + wb);
    const int32_t n_act = lower_bound_key(keys, n, (int64_t)p.ksent);
    int64_t jlo, jhi;                       // candidate centre bins
    if (p.uncut) { jlo = INT64_MIN / 2; jhi = INT64_MAX / 2; }
    else { jlo = w0 - p.cb_ceil - 2; jhi = w1 - 1 + p.cb_ceil + 2; }
    TileRange r;
    r.A0 = p.uncut ? 0 : lower_bound_key(keys, n_act, jlo - p.kmin);
    r.A1 = p.uncut ? n_act : lower_bound_key(keys, n_act, jhi + 1 - p.kmin);
    // left of the tile: the extent must reach the tile's last bin (jc >= jLmin)
    const int64_t jLmin = p.uncut ? INT64_MIN / 2 : w1 - p.cb_floor;
    int64_t jLfar = min(left_bound((double)w0, p.kappa1, p.numin_bins), w0 - 1 - mind);
    int64_t jLmid = min(left_bound((double)w0, p.kappa2, p.numin_bins), w0 - 1 - mind);
    // right of the tile: the extent must reach the tile's first bin (jc <= jRmax)
    const int64_t jRmax = p.uncut ? INT64_MAX / 2 : w0 + p.cb_floor - 2;
    int64_t jRfar = max(right_bound((double)(w1 - 1), p.kappa1, p.numin_bins), w1 - 1 + mind);
    int64_t jRmid = max(right_bound((double)(w1 - 1), p.kappa2, p.numin_bins), w1 - 1 + mind);
    if (p.mode == 1) { jLfar = jLmid = INT64_MIN / 2; jRfar = jRmid = INT64_MAX / 2; }
    if (p.mode == 2) { jLfar = INT64_MIN / 2; jRfar = INT64_MAX / 2; }
    int32_t fl0 = lower_bound_key(keys, n_act, jLmin - p.kmin);
    int32_t fl1 = lower_bound_key(keys, n_act, jLfar + 1 - p.kmin);
    int32_t ml1 = lower_bound_key(keys, n_act, jLmid + 1 - p.kmin);
    int32_t mr0 = lower_bound_key(keys, n_act, jRmid - p.kmin);
    int32_t fr0 = lower_bound_key(keys, n_act, jRfar - p.kmin);
    int32_t fr1 = lower_bound_key(keys, n_act, jRmax + 1 - p.kmin);
    // make the sequence monotone inside [A0, A1]; every adjustment only shrinks an interior class
    fl0 = min(max(fl0, r.A0), r.A1);
    fl1 = min(max(fl1, fl0), r.A1);
    ml1 = min(max(ml1, fl1), r.A1);
    fr1 = max(min(fr1, r.A1), ml1);
    fr0 = max(min(fr0, fr1), ml1);
    mr0 = max(min(mr0, fr0), ml1);
    r.FL0 = fl0; r.FL1 = fl1; r.ML1 = ml1; r.MR0 = mr0; r.FR0 = fr0; r.FR1 = fr1;
    tr[wt] = r;
    const unsigned long long nb = (unsigned long long)(w1 - w0);
    const unsigned long long nfar = (unsigned long long)(fl1 - fl0) + (unsigned long long)(fr1 - fr0);
    const unsigned long long nmid = (unsigned long long)(ml1 - fl1) + (unsigned long long)(fr0 - mr0);
    const unsigned long long nall = (unsigned long long)(r.A1 - r.A0);
    if (nfar) atomicAdd(&st->pairs_far, nfar * nb);
    if (nmid) atomicAdd(&st->pairs_mid, nmid * nb);
    if (nall > nfar + nmid) atomicAdd(&st->pairs_near, (nall - nfar - nmid) * nb);
}

// Per CTA tile: number of line chunks over the union of its warp tiles' candidates.
__global__ void __launch_bounds__(256) unit_kernel(Params p, const TileRange* __restrict__ tr, int32_t* __restrict__ counts)
{
    int ct = blockIdx.x * blockDim.x + threadIdx.x;
    if (ct >= p.n_ct) return;
    int64_t len = (int64_t)tr[ct].A1 - tr[ct].A0;
    counts[ct] = len > 0 ? (int32_t)((len + p.chunk - 1) / p.chunk) : 0;
}

}  // namespace hk
