// hk_preprocess.cuh -- steps a1-a3 of the hot path:
//   line_kernel   : per-line S, Gamma_L, alpha_D, centre bin, extent, sort key   (Eq. 5, 9, 13; L236-239)
//   gather_kernel : permute records into centre-bin order, apply the launch scale
//   range_kernel  : per level-0 tile, the candidate line range and its split into classes (L347), work-unit counts
//   node_range_kernel : per (level, tile) of the node hierarchy, the line ranges evaluated at its nodes
#pragma once
#include "hk_device.cuh"

namespace hk {

constexpr int kMaxIso = 16;               // isotopologues per species (HITRAN-style inputs)

// extra per-line arrays of HITRAN-style inputs (all null for ExoMol-style lists)
struct LineExtra {
    const double* gam_self;
    const double* delta;
    const int32_t* iso;
};

struct Params {
    // grid
    double numin, dnu;
    double inv_dnu;       // 1/dnu: for the quantities that end up in fp32 records (the integer extents use true divisions)
    int64_t N;
    // conditions folded into constants (host, fp64)
    double c2_over_T;     // h c / (k_B T)
    double tfac;          // T_ref / T
    double ln_tfac;       // ln(T_ref / T)
    double P_atm;
    double beta;          // sqrt(2 k_B T / m) / c     (alpha_D = beta nu0)
    double sfac;          // 1 / (8 pi c m Q)
    double cKfac;         // sfac / (beta sqrt(pi)): S / (alpha_D sqrt(pi)) = A g' cKfac e^(-c2 E/T) (1 - e^(-c2 nu0/T)) / nu0^3
    double inv4pic;       // 1 / (4 pi c)
    // HITRAN-style inputs (n_iso > 0): Eq. 4 self pressure, per-isotopologue beta and abundance / (8 pi c m Q)
    double P_self;
    int32_t n_iso;
    double beta_iso[kMaxIso], sfac_iso[kMaxIso], cKfac_iso[kMaxIso];
    // cut
    double cut;           // cm^-1 (ignored when uncut)
    int uncut;
    // cutting length per line (L239): 0 fixed (cut), 1 cut_factor x Gamma_L, 2 cut_factor x Gamma_D = alpha_D sqrt(ln 2).
    // Width-relative modes run in passes over classes of cutting length [cls_lo, cls_hi): a line outside the class of
    // the pass is "foreign" (not this pass's business, counted nowhere); cb_floor comes from the smallest and cb_ceil
    // from the largest cutting length of the class.
    int cut_mode;
    int count_invalid;     // count R14-skipped lines in this pass (first pass only)
    double cut_factor, cls_lo, cls_hi;
    // sort keys: key = jc - kmin in [0, ksent), ksent = sentinel for lines that contribute nothing
    int64_t kmin;
    int32_t ksent;
    int32_t compact;            // keys span [0, ksent] with ksent ~ N + 2 cut/dnu: a counting sort by key is possible
    // tile ranges
    int64_t cb_floor, cb_ceil;  // floor/ceil of cut/dnu (bins)
    double kappa1, kappa2;      // sqrt(Z1) * beta and sqrt(Z2) * beta, slightly inflated
    double kappa3;              // sqrt(ZG) * beta: beyond it no line has innermost (lane-pass) bins
    double kappaN;              // the node hierarchy takes separated tiles that lie beyond kappaN of the line: kappa2, or
                                // sqrt(HK_ZN) * beta with core_nodes (the tiles of the core outside the inner region too)
    double inv1p_kN, inv1m_kN;
    int core_nodes;             // 1: node-handled pairs may lie inside the core (|z|^2 < Z2): evaluated at the nodes with the
                                //    4-point Gauss-Hermite form ("the core at nodes")
    double inv1p_k1, inv1m_k1, inv1p_k2, inv1m_k2, inv1p_k3, inv1m_k3;   // 1/(1 + kappa), 1/(1 - kappa)
    double numin_bins;          // numin / dnu
    int32_t kb;                 // bins per lane (2, 4, 8)
    int32_t n_ct;               // tiles of 32 kb bins
    int32_t chunk;              // lines per work unit of the direct kernels
    int32_t chunk_node;         // lines per work unit of the node kernel
    int32_t chunk_centre;       // lines per work unit of the centre row kernel (a warp)
    int32_t chunk_lane;         // lines per work unit of the centre lane kernel (a CTA)
    double sep;                 // node separation: |centre - tile centre| >= sep * half-width
    int profile;                // 0 Voigt, 1 Lorentz (records carry alpha_D = 0), 2 Doppler (records carry Gamma_L = 0)
    int plinth;                 // 1: remove every line's value at the cutting length from its bins (section 2.1.1)
    double cut_bins;            // cut / dnu
    int lane_tight;             // 1: the lane-pass candidate range uses the largest z3_for(y^2) of THIS launch's lines
                                //    (0: any y -- ranges that later conditions of a batch reuse with other widths)
    int edge_nodes;             // 1: separated edge tiles go through per-bin node accumulators (edge_node_kernel)
    int mode;                   // debug: 0 default, 1 everything through the near kernel, 2 far pairs through the mid kernel,
                                //        3 direct evaluation only (no node hierarchy)
};

struct DevStats {
    unsigned long long n_skipped, n_off_grid, n_evals, n_cnt_mid, n_cnt_core;  // cnt_*: evals with |z|^2 below Z1 / Z2
    unsigned long long n_cnt_gh6, n_cnt_trap;                                  // ... below Z4 / Z3
    unsigned long long n_cnt_gh10;                                             // of n_cnt_trap: lines with y >= HK_Y10
    unsigned long long n_cnt_core_nodes;                                       // of n_cnt_core: bins of node-handled tiles (the core at nodes)
    unsigned long long n_cnt_gh10_row;                                         // of n_cnt_gh10: lines wide enough for the row kernel's 10-point class
    unsigned long long cmax_bits, cKmax_bits;                                  // max Lorentz amplitude / cK as double bits
    int32_t scale_exp;
    int32_t n_act;                                         // sorted lines with a real key (the rest carry the sentinel)
    unsigned int unit_counter_far, unit_counter_mid, unit_counter_near, unit_counter_node;
    unsigned int unit_counter_edge, unit_counter_centre, unit_counter_lane, pad2;
    unsigned long long units_far, units_mid, units_near, units_node, units_edge, units_centre;
    unsigned long long pairs_far, pairs_mid, pairs_near;   // (line, bin) slots per kernel, from the tile ranges
    unsigned long long pairs_edge, pairs_centre;
    unsigned long long pairs_edge_node;                    // (line, extent end) pairs evaluated at the nodes of their edge tile
    unsigned long long pairs_node;                         // (line, tile) pairs evaluated at nodes
    unsigned long long bins_node;                          // (line, bin) pairs those node evaluations stand for
    unsigned long long pairs_node_eval;                    // (line, tile) pairs the node kernel evaluated: must equal pairs_node
    unsigned long long pairs_node_far;                     // of pairs_node: |z|^2 >= Z1 on the whole tile (one asymptotic term)
    unsigned long long pairs_node_core;                    // of pairs_node: |z|^2 < Z2 possible on the tile (4-point form at the nodes)
    unsigned long long shift_bits;                         // max |delta P| over the lines (cm^-1) as double bits (pressure shift)
    unsigned long long n_plinth_illcond;                   // plinth removal: lines whose cutting length falls inside their core
    unsigned long long n_unsorted;                         // adjacent pairs of valid lines out of centre-bin order (input order)
    unsigned long long n_nokey;                            // lines that carry the sentinel key (invalid, off the grid, foreign)
    unsigned long long z3max_bits;                         // largest z3_for(y^2) over the lines (fp32 bits): how far innermost bins reach
    unsigned long long single_bad;                         // single-pass preprocess: lines that break its assumption (no key, or out of order)
    int32_t single_pass, pad3;                             // 1: the records of this launch were written by line_sorted_kernel
};

// What one compute leaves for the next one on the same workspace (a1/a2): a list that arrived in
// centre-bin order with every line on the grid, and the exponent of its launch scale.  A HINT, nothing more: the next
// compute writes its sorted records in one pass on the strength of it, checks both assumptions on the device while it
// does so, and runs the two-pass path after all when one of them fails.
struct DevHint {
    int32_t valid, sorted, exp, skip_two_pass;
};
constexpr int kScaleWindow = 8;      // the single pass stands when the hinted scale puts the largest amplitude within 2^(40 +- 8)

// Totals over the blocks of hk_compute_host / the class passes of a width-relative cut, kept on the device so that the
// per-block counters need no host synchronisation (read back once at the end).
struct DevTotals {
    unsigned long long n_skipped, n_off_grid, n_evals, n_plinth_illcond;
};
__global__ void add_totals_kernel(const DevStats* __restrict__ st, DevTotals* __restrict__ tot)
{
    tot->n_skipped += st->n_skipped; tot->n_off_grid += st->n_off_grid; tot->n_evals += st->n_evals;
    tot->n_plinth_illcond += st->n_plinth_illcond;
}

// The tile bounds (left_bound / right_bound) assume alpha_D = beta x centre.  With a pressure shift the profile is
// centred at nu0 + delta P while alpha_D uses the tabulated nu0 (R23), so alpha_D <= beta (centre + s) with
// s = max |delta P| over the list (found by line_kernel): the bounds stay conservative BY CONSTRUCTION when the origin
// of the wavenumber axis they see is moved down by s.  Kernels that evaluate the bounds call this first.
__device__ __forceinline__ void apply_shift_bound(Params& p, const DevStats* __restrict__ st)
{
    const double s = __longlong_as_double((long long)st->shift_bits);
    if (s > 0.0) p.numin_bins += s / p.dnu;
    // The core at nodes (core_nodes): no node-handled tile may reach into the INNER region of any line, where the profile
    // is not the smooth function the 12 nodes resolve (the Gaussian of a line with next to no Lorentz width is followed to
    // |z|^2 = 50 or HK_ZG).  z3max is the largest z3_for(y^2) of this launch's lines (line_record).
    if (p.core_nodes) {
        const float z3m = __uint_as_float((unsigned)st->z3max_bits);
        if (z3m * 1.02f > HK_ZN) {
            p.kappaN = fmin(sqrt((double)(z3m * 1.02f)) * p.beta * 1.001, p.kappa2);
            p.inv1p_kN = 1.0 / (1.0 + p.kappaN); p.inv1m_kN = 1.0 / (1.0 - p.kappaN);
        }
    }
}

__device__ __forceinline__ bool finite6(double a, double b, double c, double d, double e, double f)
{
    return isfinite(a) && isfinite(b) && isfinite(c) && isfinite(d) && isfinite(e) && isfinite(f);
}

// a / dnu, correctly rounded like the IEEE division the oracle performs, in three operations: with y = RN(1/dnu)
// (p.inv_dnu, an IEEE division on the host) and q0 = RN(a y) -- within one ulp of the quotient -- the residual
// r = a - dnu q0 is exact under FMA and RN(q0 + r y) is the correctly rounded quotient (Markstein's theorem).  A
// quotient beyond 2^62 bins (where q0 may already be infinite) is used as it is: every caller clamps it to 4e18.
__device__ __forceinline__ double div_by_dnu(const Params& p, double a)
{
    const double q0 = __dmul_rn(a, p.inv_dnu);
    const double r = __fma_rn(-p.dnu, q0, a);
    const double q1 = __fma_rn(r, p.inv_dnu, q0);
    return fabs(q0) < 4.6e18 ? q1 : q0;
}

// the bin a centre falls in, as line_math computes it (same operations, same order)
__device__ __forceinline__ int64_t centre_bin(const Params& p, double ctr)
{
    const double big = 4.0e18;
    double c = floor(div_by_dnu(p, __dsub_rn(ctr, p.numin)));
    c = fmin(fmax(c, -big), big);
    return (int64_t)c;
}

struct LineOut {
    bool valid;       // passes the R14 checks
    bool on_grid;     // extent non-empty and centre within 2^30 bins
    bool foreign;     // width-relative cut: the line's cutting length belongs to another pass
    double S, gammaL, alphaD;
    double cK;        // S / (alpha_D sqrt(pi))
    int64_t jc, ilo, ihi;
    double pos_f;     // (nu0-numin)/dnu - jc
    double shift;     // |delta P|, cm^-1 (0 without pressure shift)
};

// The fp64 arithmetic of step a1.  Extents use IEEE operations in exactly the order
// SURVEY.md 8(c).4 states (no contraction: explicit _rn intrinsics).
// gs, dl, iso: gamma_self, pressure shift and isotopologue index of HITRAN-style inputs (ignored when p.n_iso == 0)
__device__ __forceinline__ LineOut line_math(const Params& p, double nu0, double A, double g, double E,
                                             double gam, double nx, double gs = 0.0, double dl = 0.0, int32_t iso = 0)
{
    LineOut o;
    o.valid = finite6(nu0, A, g, E, gam, nx) && nu0 > 0.0 && A >= 0.0;
    if (p.n_iso > 0) o.valid = o.valid && isfinite(gs) && isfinite(dl) && iso >= 0 && iso < p.n_iso;

    o.on_grid = false;
    o.foreign = false;
    o.S = o.gammaL = o.alphaD = o.cK = 0.0;
    o.jc = 0; o.ilo = 0; o.ihi = -1; o.pos_f = 0.0; o.shift = 0.0;
    if (!o.valid) return o;
    double ctr = nu0;                                                          // centre of the profile and of the extent
    // Eq. 9 (L127) with one reciprocal: S = A g' sfac w / nu0^2 and S / (alpha_D sqrt(pi)) = A g' cKfac w / nu0^3,
    // w = e^(-c2 E/T) (1 - e^(-c2 nu0/T)); 1 - e^-x through expm1 only where the difference would cancel (x < 1)
    const double inv_nu = 1.0 / nu0;
    const double xs = p.c2_over_T * nu0;
    const double stim = xs < 1.0 ? -expm1(-xs) : 1.0 - exp(-xs);
    const double w = A * g * (inv_nu * inv_nu) * exp(-p.c2_over_T * E) * stim;
    if (p.n_iso > 0) {
        // Eq. 4 (L87), pressure shift (L238, Table 4), isotopologue table (L371-373); R23, R24
        o.alphaD = p.beta_iso[iso] * nu0;
        o.gammaL = A * p.inv4pic + exp(nx * p.ln_tfac) * (gam * (p.P_atm - p.P_self) + gs * p.P_self);
        o.S = w * p.sfac_iso[iso];
        o.cK = w * inv_nu * p.cKfac_iso[iso];
        ctr = __dadd_rn(nu0, __dmul_rn(dl, p.P_atm));                          // two roundings, as the oracle (no FMA contraction)
        o.shift = fabs(ctr - nu0);
    } else {
    o.alphaD = p.beta * nu0;                                                   // Eq. 13 (L203)
    o.gammaL = A * p.inv4pic + gam * exp(nx * p.ln_tfac) * p.P_atm;            // Eq. 5 (L91): (T_ref/T)^n = e^(n ln(T_ref/T))
    o.S = w * p.sfac;                                                          // Eq. 9 (L127)
    o.cK = w * inv_nu * p.cKfac;
    }
    // (a width or strength that overflows fp64 -- finite fields, absurd exponents -- is treated like a non-finite
    //  field, R14: the line is skipped)
    if (!isfinite(o.gammaL) || !isfinite(o.S) || !isfinite(o.cK)) { o.valid = false; o.S = o.gammaL = o.alphaD = o.cK = 0.0; return o; }
    const double big = 4.0e18;
    nu0 = ctr;
    double pos = div_by_dnu(p, __dsub_rn(nu0, p.numin));
    double c = floor(pos);
    c = fmin(fmax(c, -big), big);
    o.jc = (int64_t)c;
    o.pos_f = pos - c;
    if (!p.uncut) {
        double cutl = p.cut;
        if (p.cut_mode != 0) {                                                  // L239, R25
            cutl = p.cut_factor * (p.cut_mode == 1 ? o.gammaL : o.alphaD * 0.83255461115769775635);   // sqrt(ln 2)
            if (!(cutl > 0.0)) return o;                                        // zero width: no extent
            if (!(cutl >= p.cls_lo && cutl < p.cls_hi)) { o.foreign = true; return o; }
        }
        double lo = ceil(div_by_dnu(p, __dsub_rn(__dsub_rn(nu0, cutl), p.numin)));
        double hi = floor(div_by_dnu(p, __dsub_rn(__dadd_rn(nu0, cutl), p.numin)));
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

struct LineCounters {
    unsigned long long skipped, off, evals, cmaxb, cKmaxb, shiftb, nokey, z3b;
};

// The unsorted record and the key of one line from its fp64 parameters; flo_v: low part of the sub-bin offset (binned
// Gaussian only, R26).  Lines that contribute nothing keep the sentinel key and an empty extent.
__device__ __forceinline__ int32_t line_record(const Params& p, const LineOut& o, RecU& r, float& flo_v, LineCounters& c)
{
    int32_t k = p.ksent;
    flo_v = 0.f;
    r.jc = 0; r.f = 0.f; r.G2 = 0.f; r.a2 = 0.f; r.ilo = 0; r.ihi = -1; r.cK = 0.0;
    if (!o.valid) {
        if (p.count_invalid) ++c.skipped;
    } else if (o.foreign) {
        // belongs to another pass
    } else if (!o.on_grid) {
        ++c.off;
        r.jc = (int32_t)max(min(o.jc, (int64_t)INT32_MAX), (int64_t)INT32_MIN);
    } else {
        double Gb = o.gammaL * p.inv_dnu, ab = o.alphaD * p.inv_dnu;   // the record keeps the TRUE widths (the scatter applies the profile)
        r.jc = (int32_t)o.jc;
        // sub-bin offset relative to the NEAREST grid point, in [-1/2, 1/2]: the profile is sampled at grid points, so
        // a centre that (almost) coincides with one needs its tiny offset at full relative precision (a narrow
        // Lorentzian sampled at its peak).  Negative (sign bit set, -0 included): the nearest point is jc + 1.
        const double fd = o.pos_f > 0.5 ? o.pos_f - 1.0 : o.pos_f;
        r.f = (float)fd;
        flo_v = (float)(fd - (double)r.f);
        r.G2 = (float)(Gb * Gb);
        r.a2 = (float)(ab * ab);
        r.ilo = (int32_t)o.ilo;
        r.ihi = (int32_t)o.ihi;
        r.cK = o.cK;                                                // S/(alpha_D sqrt(pi))
        const bool gauss = p.profile == HK_PROFILE_DOPPLER || p.profile == HK_PROFILE_BINNED_GAUSSIAN;
        double cl = gauss ? 0.0 : o.S * Gb * (p.inv_dnu * 0.31830988618379067154);   // Lorentz amplitude in bin units, S Gb/(pi dnu) (none for a Gaussian)
        k = (int32_t)(o.jc - p.kmin);
        c.cmaxb = max(c.cmaxb, (unsigned long long)__double_as_longlong(cl));
        c.cKmaxb = max(c.cKmaxb, (unsigned long long)__double_as_longlong(r.cK));
        c.evals += (unsigned long long)(o.ihi - o.ilo + 1);
        c.shiftb = max(c.shiftb, (unsigned long long)__double_as_longlong(o.shift));
        // (y^2 exactly as write_sorted_records forms it)
        const float y2f = (gauss || !(r.a2 > 0.f)) ? 0.f : __fdiv_rn(r.G2, r.a2);
        // (a damping too small for the Lorentzian wing to outweigh the Gaussian at |x| = 7 counts as none: HK_ZG)
        c.z3b = max(c.z3b, (unsigned long long)__float_as_uint(y2f < 1.0e-30f ? HK_ZG : z3_for(y2f)));
        // (the per-region evaluation counts are reporting only: region_stats_kernel derives them from the records when
        //  hk_get_stats asks, so the fp64 pipe of this kernel is spent on the physics alone)
    }
    if (k == p.ksent) ++c.nokey;
    return k;
}

// block reduction of the per-line counters: sums and maxima (positive doubles order as their bit patterns)
__device__ __forceinline__ void reduce_line_counters(const LineCounters& c, unsigned long long bad, DevStats* __restrict__ st)
{
    __shared__ unsigned long long sh[9][8];
    unsigned long long v[9] = {c.skipped, c.off, c.evals, c.nokey, bad, c.cmaxb, c.cKmaxb, c.shiftb, c.z3b};
#pragma unroll
    for (int q = 0; q < 9; ++q) {
        unsigned long long x = v[q];
        for (int o = 16; o > 0; o >>= 1) {
            unsigned long long y = __shfl_xor_sync(0xffffffffu, x, o);
            x = (q < 5) ? x + y : max(x, y);
        }
        if ((threadIdx.x & 31) == 0) sh[q][threadIdx.x >> 5] = x;
    }
    __syncthreads();
    if (threadIdx.x < 9) {
        int q = threadIdx.x;
        unsigned long long x = sh[q][0];
        for (int w = 1; w < 8; ++w) x = (q < 5) ? x + sh[q][w] : max(x, sh[q][w]);
        unsigned long long* dst = q == 0 ? &st->n_skipped : q == 1 ? &st->n_off_grid : q == 2 ? &st->n_evals
                                : q == 3 ? &st->n_nokey : q == 4 ? &st->single_bad
                                : q == 5 ? &st->cmax_bits : q == 6 ? &st->cKmax_bits : q == 7 ? &st->shift_bits : &st->z3max_bits;
        if (x) { if (q < 5) atomicAdd(dst, x); else atomicMax(dst, x); }
    }
}

// The six fp64 fields of the lines kAhead iterations AHEAD travel global -> shared with cp.async (8 B per field per
// thread, no registers held) while the current line's exponentials and divisions run: every thread reads back only
// what it copied itself, so cp.async.wait_group is all the synchronisation there is.
__device__ __forceinline__ void cp_async8(double* smem_dst, const double* gsrc)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((uint32_t)__cvta_generic_to_shared(smem_dst)), "l"(gsrc) : "memory");
}
constexpr int kAhead = 2;
struct LineStage {
    double (*stage)[6][256];                     // [kAhead + 1][6][256] in shared memory
    const double* src[6];
    int buf;
    __device__ __forceinline__ void issue(int slot, int64_t i, int64_t n) const
    {
        if (i < n) {
#pragma unroll
            for (int q = 0; q < 6; ++q) cp_async8(&stage[slot][q][threadIdx.x], src[q] + i);
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    }
    __device__ __forceinline__ void prime(int64_t i, int64_t stride, int64_t n)
    {
        buf = 0;
#pragma unroll
        for (int a = 0; a < kAhead; ++a) issue(a, i + a * stride, n);
    }
    // start the copy for iteration i + kAhead strides, wait for iteration i's
    __device__ __forceinline__ void step(int64_t i, int64_t stride, int64_t n) const
    {
        issue(buf == 0 ? kAhead : buf - 1, i + kAhead * stride, n);     // slot (buf + kAhead) mod (kAhead + 1)
        asm volatile("cp.async.wait_group %0;" ::"n"(kAhead) : "memory");
    }
    __device__ __forceinline__ double get(int q) const { return stage[buf][q][threadIdx.x]; }
    __device__ __forceinline__ void next() { buf = (buf == kAhead) ? 0 : buf + 1; }
    __device__ __forceinline__ void drain() const { asm volatile("cp.async.wait_group 0;" ::: "memory"); }
};

__global__ void __launch_bounds__(256, 4) line_kernel(Params p, const double* __restrict__ nu0,
                                                   const double* __restrict__ A, const double* __restrict__ g,
                                                   const double* __restrict__ E, const double* __restrict__ gam,
                                                   const double* __restrict__ nx, LineExtra ex, int64_t n,
                                                   RecU* __restrict__ rec, int32_t* __restrict__ key,
                                                   int32_t* __restrict__ idx, float* __restrict__ flo,
                                                   int32_t* __restrict__ hist, DevStats* __restrict__ st,
                                                   const DevHint* __restrict__ hint)
{
    // idx: identity permutation for the radix sort (null with the counting sort); hist: the counting sort's buckets (null
    // otherwise) -- the histogram of the keys rides along here, its atomics hidden under the fp64 arithmetic: lanes of a
    // warp with equal keys (neighbours, in a list that arrives sorted) are served by ONE atomic.
    // hint (nullable): the single pass (line_sorted_kernel) has done this launch's work already
    if (hint && hint->skip_two_pass) return;
    __shared__ double stage[kAhead + 1][6][256];
    LineStage ls = {stage, {nu0, A, g, E, gam, nx}, 0};
    LineCounters c = {0, 0, 0, 0, 0, 0, 0, 0};
    const int64_t n_round = hist ? ((n + 31) & ~31LL) : n;                   // (warp-uniform trip count for the match)
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    ls.prime(i, stride, n);
    for (; i < n_round; i += stride, ls.next()) {
        ls.step(i, stride, n);
        int32_t k = -1;                         // (lanes past the end of the list take part in the match only)
        if (i < n) {
            LineOut o = p.n_iso > 0 ? line_math(p, ls.get(0), ls.get(1), ls.get(2), ls.get(3), ls.get(4), ls.get(5),
                                                ex.gam_self[i], ex.delta[i], ex.iso[i])
                                    : line_math(p, ls.get(0), ls.get(1), ls.get(2), ls.get(3), ls.get(4), ls.get(5));
            RecU r;
            float flo_v;
            k = line_record(p, o, r, flo_v, c);
            if (flo) flo[i] = flo_v;
            rec[i] = r;
            key[i] = k;
            if (idx) idx[i] = (int32_t)i;
        }
        if (hist) {
            const unsigned peers = __match_any_sync(0xffffffffu, k);
            if (k >= 0 && (int)(threadIdx.x & 31) == __ffs(peers) - 1) atomicAdd(hist + k, __popc(peers));
        }
    }
    ls.drain();
    reduce_line_counters(c, 0ULL, st);
}

// Per-region evaluation counts (hk_stats.n_evals_far / mid / core / gh6 / trap / gh10) from the sorted records of the
// last compute: for each line the number of bins of its extent with |z|^2 below each threshold.  Run on demand.
__global__ void __launch_bounds__(256) region_stats_kernel(const float4* __restrict__ recA, const float4* __restrict__ recB,
                                                           int64_t n, int profile, int kb, DevStats* __restrict__ st)
{
    unsigned long long c[6] = {0, 0, 0, 0, 0, 0};        // below Z1, Z2, Z4, Z3 (trapezoid region), of that with y >= HK_Y10, of that in rows
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const float4 ra = recA[i], rb = recB[i];
        const int32_t ilo = __float_as_int(rb.y), ihi = __float_as_int(rb.z);
        if (ihi < ilo) continue;
        const bool gauss = profile == HK_PROFILE_DOPPLER || profile == HK_PROFILE_BINNED_GAUSSIAN;
        // (recA.z: G2, or the low part of the offset for the binned Gaussian; recB.x: a2, 0 for a pure Lorentzian)
        const double G2 = gauss ? 0.0 : (double)ra.z, a2 = (double)rb.x;
        const double pos = (double)__float_as_int(ra.x) + (double)ra.y;      // nearest grid point + offset in [-1/2, 1/2]
        const double y2 = a2 > 0.0 ? G2 / a2 : 1.0e300;
        const double z3 = (double)z3_for((float)fmin(y2, 1.0e30)), z4 = fmax((double)z4_for((float)fmin(y2, 1.0e30)), z3);
        const double t[4] = {(double)HK_Z1 * a2 - G2, (double)HK_Z2 * a2 - G2, z4 * a2 - G2, z3 * a2 - G2};
#pragma unroll
        for (int q = 0; q < 4; ++q)
            c[q] += (unsigned long long)count_within(pos, t[q] > 0 ? (double)sqrtf((float)t[q]) : 0.0, ilo, ihi);
        if (y2 >= (double)(HK_Y10 * HK_Y10)) {
            const unsigned long long c10 = (unsigned long long)count_within(pos, t[3] > 0 ? (double)sqrtf((float)t[3]) : 0.0, ilo, ihi);
            c[4] += c10;
            // the row kernel evaluates these bins itself (class R10) when alpha_D >= 0.85 bins per 64 bins of tile (centre_setup)
            if (a2 > 0.0 && 1.0 / sqrt(a2) < 1.0 / (0.85 * (double)(kb / 2))) c[5] += c10;
        }
    }
#pragma unroll
    for (int q = 0; q < 6; ++q) {
        unsigned long long x = c[q];
        for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
        if ((threadIdx.x & 31) == 0 && x) {
            unsigned long long* dst = q == 0 ? &st->n_cnt_mid : q == 1 ? &st->n_cnt_core : q == 2 ? &st->n_cnt_gh6
                                    : q == 3 ? &st->n_cnt_trap : q == 4 ? &st->n_cnt_gh10 : &st->n_cnt_gh10_row;
            atomicAdd(dst, x);
        }
    }
}

// Power-of-two launch scale from the maxima (max Lorentz amplitude -> 2^40, and cK kept below 2^100), DESIGN.md
// section 4 "dynamic range".
__device__ __forceinline__ int scale_exp_of(const DevStats* st)
{
    double cmax = __longlong_as_double((long long)st->cmax_bits);
    double cKmax = __longlong_as_double((long long)st->cKmax_bits);
    int e = 0;
    if (cmax > 0.0 && isfinite(cmax)) e = 40 - ilogb(cmax);
    if (cKmax > 0.0 && isfinite(cKmax)) e = min(e, 100 - ilogb(cKmax));
    // no Lorentz amplitude at all (Doppler / binned Gaussian): the largest Gaussian amplitude goes to 2^100, which leaves
    // 226 binades below it -- exp(-x^2) is followed down to x^2 = HK_ZG (gauss_term, hk_device.cuh)
    if (!(cmax > 0.0) && cKmax > 0.0 && isfinite(cKmax)) e = 100 - ilogb(cKmax);
    return max(-900, min(900, e));
}

// One thread, after line_kernel (two-pass path).
__global__ void scale_kernel(DevStats* st, const DevHint* __restrict__ hint)
{
    if (hint && hint->skip_two_pass) return;
    st->scale_exp = scale_exp_of(st);
}

// One thread, after line_sorted_kernel: did the single pass stand?  It does when it ran at all (the hint said "sorted"),
// met no line without a key and no pair out of order, and the hinted scale is within kScaleWindow binades of the scale
// this launch's own maxima ask for.  Otherwise the counters it left are cleared and the two-pass path runs.
__global__ void single_pass_decide_kernel(DevStats* st, DevHint* hint)
{
    const bool ran = hint->valid && hint->sorted;
    const int e = scale_exp_of(st);
    const bool ok = ran && st->single_bad == 0ULL && abs(e - hint->exp) <= kScaleWindow;
    hint->skip_two_pass = ok ? 1 : 0;
    st->single_pass = ok ? 1 : 0;
    if (ok) { st->scale_exp = hint->exp; return; }
    st->n_skipped = st->n_off_grid = st->n_evals = st->n_nokey = st->single_bad = 0ULL;
    st->cmax_bits = st->cKmax_bits = st->shift_bits = st->z3max_bits = 0ULL;
}

// One thread, after the records are in place (either path): what this launch knows, for the next one.
__global__ void hint_update_kernel(const DevStats* __restrict__ st, DevHint* hint)
{
    hint->exp = scale_exp_of(st);
    hint->sorted = st->single_pass ? 1 : (st->n_unsorted == 0ULL && st->n_nokey == 0ULL ? 1 : 0);
    hint->valid = 1;
}

// The sorted records of one line (recA, recB, recN, recC at position `pos`) from its unsorted record.
__device__ __forceinline__ void write_sorted_records(const RecU& r, float flo_v, bool have_flo, double scale, int profile, int64_t pos,
                                                     float4* __restrict__ recA, float4* __restrict__ recB,
                                                     float4* __restrict__ recN, float4* __restrict__ recC)
{
    float cK = (float)(r.cK * scale);                              // scale = 2^scale_exp: exact
    // c = cK * G a / sqrt(pi)  (Lorentz amplitude S Gamma_L/(pi dnu^2) in bin units)
    const bool gauss = profile == HK_PROFILE_DOPPLER || profile == HK_PROFILE_BINNED_GAUSSIAN;
    float G2 = gauss ? 0.f : r.G2;
    float c = cK * sqrtf(G2 * r.a2) * 0.564189583547756f;
    // a Lorentzian of zero (or fp32-denormal) width contributes nothing anywhere but would give 0/0 on a grid point
    // it coincides with: keep it out with c = 0 and a harmless width
    if (profile == HK_PROFILE_LORENTZ && !(G2 >= 1.0e-30f)) { G2 = 1.0f; c = 0.f; }
    // a pure Lorentzian is what every formula of the accumulation kernels reduces to at alpha_D = 0 (no core,
    // no second asymptotic term); a pure Gaussian is the Voigt function at Gamma_L = 0 (c = 0: no wings)
    const float a2 = profile == HK_PROFILE_LORENTZ ? 0.f : r.a2;
    const bool up = signbit(r.f);                                  // centre = (jc + 1) + f with f <= 0
    // (binned Gaussian: G2 = 0 and c = 0 everywhere, and the free slot carries the low part of the sub-bin offset)
    recA[pos] = make_float4(__int_as_float(r.jc + (up ? 1 : 0)), r.f, (have_flo && profile == HK_PROFILE_BINNED_GAUSSIAN) ? flo_v : G2, c);
    recB[pos] = make_float4(a2, __int_as_float(r.ilo), __int_as_float(r.ihi), cK);
    // node record: offset from jc in [0, 1) rounded to the nearest 1/8192 (|error| <= 2^-14 bins; 8192 clamps to 8191),
    // a2 rounded to nearest at 11 mantissa bits (|error| <= 2^-12 relative, unbiased)
    const uint32_t f13 = min(8191u, (uint32_t)__float2int_rn((up ? 1.0f + r.f : r.f) * 8192.0f));
    const uint32_t a19 = (((uint32_t)__float_as_int(a2) + 0x800u) >> 12) & 0x7FFFFu;
    recN[pos] = make_float4(__int_as_float(r.jc), __int_as_float((int)((f13 << 19) | a19)), G2, c);
    // the per-line part of the centre kernels (hk_centre.cuh): IEEE roots and quotients, once per line.
    // ip = 1/(cK y), the reciprocal amplitude of the Gauss-Hermite rows; 0: no such rows (G = 0, or an amplitude
    // below the range of the launch)
    float inva = 0.f, y2 = 0.f, ip = 0.f;
    if (a2 > 0.f) {
        inva = __fsqrt_rn(__fdiv_rn(1.0f, a2));          // the Gaussian tail amplifies an error of x by 2 x^2
        y2 = gauss ? 0.f : __fdiv_rn(G2, a2);
        const float P = cK * __fsqrt_rn(y2);
        if (P > 1.0e-30f && c != 0.f) ip = __fdiv_rn(1.0f, P);
    }
    recC[pos] = make_float4(inva, __fmul_rn(-r.f, inva), y2, ip);
}

// ---- single-pass preprocess (steps a1 + a2 in one kernel) -----------------------------------------------------------
// Line lists are stored in wavenumber order, and conditions change little from one call to the next.  When the previous
// compute on this workspace saw a list in centre-bin order with every line on the grid (DevHint), the sorted position of
// line i is i, and with the previous launch scale as a stand-in for this one the fp32 records can be written as the
// fp64 parameters are formed: no unsorted record, no key array, no histogram, no scatter.  Both assumptions are CHECKED
// here (single_bad counts lines without a key and adjacent pairs out of order; the maxima give this launch's own
// scale) and single_pass_decide_kernel discards the result when one fails.  Same fp64 arithmetic (line_math,
// line_record) and same record arithmetic (write_sorted_records) as the two-pass path.
__global__ void __launch_bounds__(256, 3) line_sorted_kernel(Params p, const double* __restrict__ nu0,
                                                          const double* __restrict__ A, const double* __restrict__ g,
                                                          const double* __restrict__ E, const double* __restrict__ gam,
                                                          const double* __restrict__ nx, LineExtra ex, int64_t n,
                                                          const DevHint* __restrict__ hint, DevStats* __restrict__ st,
                                                          int32_t* __restrict__ key_sorted, int32_t* __restrict__ idx_sorted,
                                                          float4* __restrict__ recA, float4* __restrict__ recB,
                                                          float4* __restrict__ recN, float4* __restrict__ recC)
{
    if (!(hint->valid && hint->sorted)) return;
    __shared__ double stage[kAhead + 1][6][256];
    LineStage ls = {stage, {nu0, A, g, E, gam, nx}, 0};
    const double scale = scalbn(1.0, hint->exp);
    const int lane = threadIdx.x & 31;
    LineCounters c = {0, 0, 0, 0, 0, 0, 0, 0};
    unsigned long long bad = 0;
    const int64_t n_round = (n + 31) & ~31LL;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    ls.prime(i, stride, n);
    for (; i < n_round; i += stride, ls.next()) {
        ls.step(i, stride, n);
        const bool live = i < n;
        int64_t jc = INT64_MAX;                  // (lanes past the end: never "before" their neighbour)
        RecU r;
        int32_t k = p.ksent;
        if (live) {
            LineOut o = p.n_iso > 0 ? line_math(p, ls.get(0), ls.get(1), ls.get(2), ls.get(3), ls.get(4), ls.get(5),
                                                ex.gam_self[i], ex.delta[i], ex.iso[i])
                                    : line_math(p, ls.get(0), ls.get(1), ls.get(2), ls.get(3), ls.get(4), ls.get(5));
            float flo_v;
            k = line_record(p, o, r, flo_v, c);
            jc = o.jc;
            if (k == p.ksent) ++bad;
        }
        // in order?  against the line before (lane 0: that line's centre bin again, from its wavenumber)
        int64_t prev = __shfl_up_sync(0xffffffffu, jc, 1);
        if (lane == 0) {
            prev = jc;
            if (live && i > 0) {
                double ctr = nu0[i - 1];
                if (p.n_iso > 0) ctr = __dadd_rn(ctr, __dmul_rn(ex.delta[i - 1], p.P_atm));
                prev = centre_bin(p, ctr);
            }
        }
        if (!live) continue;
        if (jc < prev) ++bad;
        key_sorted[i] = k;
        idx_sorted[i] = (int32_t)i;
        write_sorted_records(r, 0.f, false, scale, p.profile, i, recA, recB, recN, recC);
    }
    ls.drain();
    reduce_line_counters(c, bad, st);
}

// Permute by the index array of a sort (CUB path, and the later conditions of a batch, which reuse the order).
__global__ void __launch_bounds__(256) gather_kernel(const RecU* __restrict__ rec, const int32_t* __restrict__ idx_sorted,
                                                     const float* __restrict__ flo, int64_t n,
                                                     const DevStats* __restrict__ st,
                                                     float4* __restrict__ recA, float4* __restrict__ recB,
                                                     float4* __restrict__ recN, float4* __restrict__ recC, int profile)
{
    const double scale = scalbn(1.0, st->scale_exp);
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const int32_t src = idx_sorted[i];
        write_sorted_records(rec[src], flo ? flo[src] : 0.f, flo != nullptr, scale, profile, i, recA, recB, recN, recC);
    }
}

// ---- counting sort by centre bin (step a2 when the keys are compact: any fixed cut) --------------------------------
// Only the GROUPING by key matters to the accumulation kernels (their line ranges are key ranges), not the order inside
// a key.  So: histogram of the keys (in line_kernel) -> exclusive scan -> every line takes the next free slot of its key's bucket and
// writes its sorted records there, straight from the unsorted record (the gather is the scatter).  Lanes of a warp
// with equal keys -- neighbours, in a list that arrives sorted -- are served by ONE atomic.  A list that is already
// in order costs one streaming pass; nothing is decided on the host.
__global__ void __launch_bounds__(256) scatter_kernel(const RecU* __restrict__ rec, const int32_t* __restrict__ key,
                                                      const float* __restrict__ flo, int64_t n, int32_t* __restrict__ cursor,
                                                      DevStats* __restrict__ st, int32_t* __restrict__ key_sorted,
                                                      int32_t* __restrict__ idx_sorted, float4* __restrict__ recA,
                                                      float4* __restrict__ recB, float4* __restrict__ recN,
                                                      float4* __restrict__ recC, int profile,
                                                      const DevHint* __restrict__ hint)
{
    if (hint && hint->skip_two_pass) return;
    const double scale = scalbn(1.0, st->scale_exp);
    const int lane = threadIdx.x & 31;
    const unsigned lt_mask = (1u << lane) - 1u;
    const int64_t n_round = (n + 31) & ~31LL;
    unsigned long long unsorted = 0;             // adjacent pairs out of key order in the caller's list (hk_stats.n_unsorted)
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n_round; i += (int64_t)gridDim.x * blockDim.x) {
        const bool live = i < n;
        const int32_t k = live ? key[i] : -1;
        int32_t prev = __shfl_up_sync(0xffffffffu, k, 1);
        if (lane == 0) prev = (live && i > 0) ? key[i - 1] : k;
        if (live && i > 0 && k < prev) ++unsorted;
        const unsigned peers = __match_any_sync(0xffffffffu, k);
        const int leader = __ffs(peers) - 1;
        int32_t base = 0;
        if (live && lane == leader) base = atomicAdd(cursor + k, __popc(peers));
        base = __shfl_sync(0xffffffffu, base, leader);
        if (!live) continue;
        const int64_t pos = (int64_t)base + __popc(peers & lt_mask);
        key_sorted[pos] = k;
        idx_sorted[pos] = (int32_t)i;
        write_sorted_records(rec[i], flo ? flo[i] : 0.f, flo != nullptr, scale, profile, pos, recA, recB, recN, recC);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) unsorted += __shfl_xor_sync(0xffffffffu, unsorted, o);
    if (lane == 0 && unsorted) atomicAdd(&st->n_unsorted, unsorted);
}

// ---- batched conditions that differ in PRESSURE only (hk_compute_batch, the paper's "multiple pressure points") ------
// With T, Q and the mass unchanged, the strength, the Doppler width, the centre bin, the extent and the order of the
// lines -- and with them the tile and node ranges -- are those of the previous condition; only Gamma_L moves.  One
// streaming pass over the SORTED records puts the new (Gamma_L/dnu)^2 and what follows from it (Lorentz amplitude, y^2,
// 1/(cK y)) in place, from the same fp64 expression line_kernel uses (Eq. 5), read through the sort's permutation.
__global__ void __launch_bounds__(256) rewidth_kernel(Params p, const double* __restrict__ A, const double* __restrict__ gam,
                                                      const double* __restrict__ nx, const int32_t* __restrict__ idx_sorted,
                                                      const DevStats* __restrict__ st, float4* __restrict__ recA,
                                                      const float4* __restrict__ recB, float4* __restrict__ recN,
                                                      float4* __restrict__ recC)
{
    const int64_t n_act = st->n_act;
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n_act; i += (int64_t)gridDim.x * blockDim.x) {
        const int32_t src = idx_sorted[i];
        const double gammaL = A[src] * p.inv4pic + gam[src] * exp(nx[src] * p.ln_tfac) * p.P_atm;      // Eq. 5 (L91), as line_math
        const double Gb = gammaL / p.dnu;
        const float G2 = (float)(Gb * Gb);
        const float4 rb = recB[i];
        const float a2 = rb.x, cK = rb.w;
        const float c = cK * sqrtf(G2 * a2) * 0.564189583547756f;
        float4 ra = recA[i], rn = recN[i], rc = recC[i];
        ra.z = G2; ra.w = c;
        rn.z = G2; rn.w = c;
        float y2 = 0.f, ip = 0.f;
        if (a2 > 0.f) {
            y2 = __fdiv_rn(G2, a2);
            const float P = cK * __fsqrt_rn(y2);
            if (P > 1.0e-30f && c != 0.f) ip = __fdiv_rn(1.0f, P);
        }
        rc.z = y2; rc.w = ip;
        recA[i] = ra; recN[i] = rn; recC[i] = rc;
    }
}

// the counters a run recounts (work-unit cursors, evaluated pairs); everything else in DevStats stays as the previous
// condition of the batch left it
__global__ void reset_run_kernel(DevStats* st)
{
    st->unit_counter_far = st->unit_counter_mid = st->unit_counter_near = st->unit_counter_node = 0u;
    st->unit_counter_edge = st->unit_counter_centre = st->unit_counter_lane = 0u;
    st->units_far = st->units_mid = st->units_near = st->units_node = st->units_edge = st->units_centre = 0ULL;
    st->pairs_node_eval = 0ULL;
    st->pairs_edge_node = 0ULL;
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
// (the reciprocals 1/(1 + kap), 1/(1 - kap) come from the host: one rounding more, far inside the margin of 3 bins)
__device__ __forceinline__ int64_t left_bound(double w0, double kap, double inv1p, double numin_bins)
{
    // pos + 1 <= (w0 - kap numin_bins) / (1 + kap)   =>   w0 - pos >= kap (numin_bins + pos)
    return (int64_t)floor((w0 - kap * (numin_bins + 1.0)) * inv1p) - 3;
}
__device__ __forceinline__ int64_t right_bound(double w1m1, double kap, double inv1m, double numin_bins)
{
    // pos >= (w1 - 1 + kap numin_bins) / (1 - kap)   =>   pos - (w1 - 1) >= kap (numin_bins + pos)
    if (!(kap < 0.9)) return INT64_MAX / 2;
    return (int64_t)ceil((w1m1 + kap * (numin_bins + 1.0)) * inv1m) + 3;
}

// Key thresholds of one tile [w0, w1) of width W (any level) for the node hierarchy.  A line with centre bin jc is
// "handled at the nodes of this tile or of an ancestor" when loL <= jc <= upL (left of the tile) or dnR <= jc <= hiR
// (right): the tile lies inside the line's extent, |z|^2 >= Z2 on all of it, and the centre is at least sep half-widths
// from the tile centre.  The sets of a parent are nested in those of its children.
struct NodeKeys {
    int64_t loL, upL, dnR, hiR;
};
constexpr int64_t kBigKey = INT64_MAX / 4;

__device__ __forceinline__ NodeKeys node_keys(const Params& p, int64_t w0, int64_t W)
{
    const int64_t w1 = min(p.N, w0 + W);
    const double m = (double)w0 + 0.5 * (double)(W - 1), h = 0.5 * (double)W;
    NodeKeys k;
    k.loL = p.uncut ? -kBigKey : w1 - p.cb_floor;
    k.hiR = p.uncut ? kBigKey : w0 + p.cb_floor - 2;
    const int64_t sepL = (int64_t)floor(m - p.sep * h) - 1;
    const int64_t sepR = (int64_t)ceil(m + p.sep * h);
    k.upL = min(sepL, left_bound((double)w0, p.kappaN, p.inv1p_kN, p.numin_bins));
    k.dnR = max(sepR, right_bound((double)(w1 - 1), p.kappaN, p.inv1m_kN, p.numin_bins));
    // empty sets are written as [lo, lo - 1] / [hi + 1, hi]
    k.upL = max(k.upL, k.loL - 1);
    k.dnR = min(k.dnR, k.hiR + 1);
    return k;
}

// Extent ends ("edges").  A tile that a line's extent covers only in part, with the line centre at least sep
// half-widths away and |z|^2 >= Z2 on all of it, is evaluated at the tile's nodes too; the node values go to per-bin
// accumulators indexed by the bin at which the extent ends and reach the bins through a prefix / suffix sum over the
// tile (edge_node_kernel).  For the tile [w0, w0 + W): a line LEFT of it (its extent ends inside
// the tile) qualifies when jc <= upL, a line RIGHT of it (its extent starts inside) when jc >= dnR.  The same
// thresholds take these lines out of the direct edge kernel's ranges in range_kernel.
struct EdgeKeys {
    int64_t upL, dnR;
};

__device__ __forceinline__ int64_t edge_key_upL(const Params& p, int64_t w0, int64_t W)
{
    const int64_t w1 = min(p.N, w0 + W);
    const int64_t mind = (int64_t)kMinDistPerKB * p.kb;
    const double m = (double)w0 + 0.5 * (double)(W - 1), h = 0.5 * (double)W;
    const int64_t sepL = (int64_t)floor(m - p.sep * h) - 1;
    const int64_t jLmid = min(left_bound((double)w0, p.kappa2, p.inv1p_k2, p.numin_bins), w0 - 1 - mind);
    // and clearly not interior: jc <= jLmin - 2 = w1 - cb_floor - 2.  (ihi = jc + floor(cut/dnu) + 0 or 1: a line with
    // jc = jLmin - 1 may cover the tile completely and end in the NEXT one, which the centre bin alone cannot tell;
    // such pairs stay with the masked direct kernel, and every pair kept here has its extent end inside this tile)
    return min(min(sepL, jLmid), w1 - p.cb_floor - 2);
}
__device__ __forceinline__ int64_t edge_key_dnR(const Params& p, int64_t w0, int64_t W)
{
    const int64_t w1 = min(p.N, w0 + W);
    const int64_t mind = (int64_t)kMinDistPerKB * p.kb;
    const double m = (double)w0 + 0.5 * (double)(W - 1), h = 0.5 * (double)W;
    const int64_t sepR = (int64_t)ceil(m + p.sep * h);
    const int64_t jRmid = max(right_bound((double)(w1 - 1), p.kappa2, p.inv1m_k2, p.numin_bins), w1 - 1 + mind);
    return max(max(sepR, jRmid), w0 + p.cb_floor);               // jc >= jRmax + 2 = w0 + cb_floor (same argument, mirrored)
}
__device__ __forceinline__ EdgeKeys edge_keys(const Params& p, int64_t w0, int64_t W)
{
    EdgeKeys k;
    k.upL = edge_key_upL(p, w0, W);
    k.dnR = edge_key_dnR(p, w0, W);
    return k;
}

// The core at nodes, counted (on demand, for hk_get_stats): for each line, the bins with |z|^2 < Z2 that lie in tiles the
// node hierarchy handles -- at level 0 or through an ancestor -- and are therefore covered by interpolation instead of
// being evaluated one by one.  The same keys as range_kernel / node_range_kernel (node_keys), per line.
__global__ void __launch_bounds__(256) core_nodes_stats_kernel(Params p, Levels lv, const float4* __restrict__ recA,
                                                               const float4* __restrict__ recB, const float4* __restrict__ recN,
                                                               int64_t n, DevStats* __restrict__ st)
{
    apply_shift_bound(p, st);
    unsigned long long moved = 0;
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const float4 ra = recA[i], rb = recB[i];
        const int64_t ilo = __float_as_int(rb.y), ihi = __float_as_int(rb.z);
        const double a2 = (double)rb.x, G2 = (double)ra.z;
        const double t2 = (double)HK_Z2 * a2 - G2;
        if (ihi < ilo || !(t2 > 0.0)) continue;
        const double R = (double)sqrtf((float)t2);                        // (as region_stats_kernel counts the core)
        const double pos = (double)__float_as_int(ra.x) + (double)ra.y;
        const int64_t jc = __float_as_int(recN[i].x);
        const int64_t b_lo = max(ilo, (int64_t)(floor(pos - R) + 1.0)), b_hi = min(ihi, (int64_t)(ceil(pos + R) - 1.0));
        const int64_t wb = lv.w0;
        for (int64_t t0 = (b_lo / wb) * wb; t0 <= b_hi; t0 += wb) {
            bool handled = false;
            for (int l = 0; l < lv.n_levels && !handled; ++l) {
                const int64_t W = wb << l;
                const NodeKeys k = node_keys(p, (t0 / W) * W, W);
                handled = (jc >= k.loL && jc <= k.upL) || (jc >= k.dnR && jc <= k.hiR);
            }
            if (handled) moved += (unsigned long long)count_within(pos, R, max(ilo, t0), min(ihi, t0 + wb - 1));
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) moved += __shfl_xor_sync(0xffffffffu, moved, o);
    if ((threadIdx.x & 31) == 0 && moved) atomicAdd(&st->n_cnt_core_nodes, moved);
}

// index of the first sorted line with centre bin >= j (keys are jc - kmin)
__device__ __forceinline__ int32_t idx_of(const Params& p, const int32_t* __restrict__ keys, int32_t n_act, int64_t j)
{
    if (j <= -kBigKey / 2) return 0;
    if (j >= kBigKey / 2) return n_act;
    return lower_bound_key(keys, n_act, j - p.kmin);
}

// One thread per (level, tile) entry: the four index ranges of lines evaluated at this tile's nodes
// ( = handled here but not by the parent), and the number of work units they make.
__global__ void __launch_bounds__(256) node_range_kernel(Params p, Levels lv, const int32_t* __restrict__ keys, int32_t n,
                                                         const TileRange* __restrict__ tr, NodeRange* __restrict__ nr,
                                                         int32_t* __restrict__ counts, DevStats* __restrict__ st)
{
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= lv.n_entries) return;
    apply_shift_bound(p, st);
    int l = 0;
    while (l + 1 < lv.n_levels && e >= lv.off[l + 1]) ++l;
    const int64_t j = e - lv.off[l];
    const int64_t W = (int64_t)lv.w0 << l;
    const int64_t w0 = j * W;
    const int32_t n_act = lower_bound_key(keys, n, (int64_t)p.ksent);
    if (e == 0) st->n_act = n_act;
    int32_t a, b, c, d;                          // handled here or above: [a, b) on the left, [c, d) on the right
    if (l == 0) {                                // the same indices the direct kernels exclude
        const TileRange t = tr[j];
        a = t.FL0; b = t.NL; c = t.NR; d = t.FR1;
    } else {
        const NodeKeys k = node_keys(p, w0, W);
        a = idx_of(p, keys, n_act, k.loL);
        b = max(a, idx_of(p, keys, n_act, k.upL + 1));
        c = idx_of(p, keys, n_act, k.dnR);
        d = max(c, idx_of(p, keys, n_act, k.hiR + 1));
    }
    int32_t pa = n_act, pb = n_act, pc = 0, pd = 0;   // the parent's sets (none at the top level)
    if (l + 1 < lv.n_levels) {
        const int64_t Wp = 2 * W;
        const NodeKeys k = node_keys(p, (j >> 1) * Wp, Wp);
        pa = idx_of(p, keys, n_act, k.loL);
        pb = max(pa, idx_of(p, keys, n_act, k.upL + 1));
        pc = idx_of(p, keys, n_act, k.dnR);
        pd = max(pc, idx_of(p, keys, n_act, k.hiR + 1));
    } else {
        pa = pb = b;                              // nothing removed: [a, min(b, pa)) = [a, b), [max(a, pb), b) empty
        pc = pd = d;
    }
    NodeRange r;
    r.a0 = a; r.a1 = max(a, min(b, pa));          // left sliver: inside this tile's reach but not the parent's
    r.b0 = min(b, max(r.a1, pb)); r.b1 = b;       // left main: closer than the parent's separation
    r.c0 = c; r.c1 = max(c, min(d, pc));          // right main
    r.d0 = min(d, max(r.c1, pd)); r.d1 = d;       // right sliver
    // where one asymptotic term suffices on the whole tile (|z|^2 >= Z1): the same bound range_kernel uses for "far"
    r.fL = idx_of(p, keys, n_act, left_bound((double)w0, p.kappa1, p.inv1p_k1, p.numin_bins) + 1);
    r.fR = idx_of(p, keys, n_act, right_bound((double)(min(p.N, w0 + W) - 1), p.kappa1, p.inv1m_k1, p.numin_bins));
    // where the two asymptotic terms do not hold on the whole tile (the core at nodes): the bound range_kernel uses for "mid"
    r.gL = r.gR = 0;
    if (p.core_nodes) {
        r.gL = idx_of(p, keys, n_act, left_bound((double)w0, p.kappa2, p.inv1p_k2, p.numin_bins) + 1);
        r.gR = idx_of(p, keys, n_act, right_bound((double)(min(p.N, w0 + W) - 1), p.kappa2, p.inv1m_k2, p.numin_bins));
    }
    nr[e] = r;
    const int64_t tot = (int64_t)(r.a1 - r.a0) + (r.b1 - r.b0) + (r.c1 - r.c0) + (r.d1 - r.d0);
    counts[e] = (int32_t)((tot + p.chunk_node - 1) / p.chunk_node);
    if (tot) {
        const int64_t nfar = (int64_t)max(0, min(r.a1, r.fL) - r.a0) + max(0, min(r.b1, r.fL) - r.b0)
                           + max(0, r.c1 - max(r.c0, r.fR)) + max(0, r.d1 - max(r.d0, r.fR));
        if (nfar) atomicAdd(&st->pairs_node_far, (unsigned long long)nfar);
        auto within = [&](int32_t x0, int32_t x1) { return (int64_t)max(0, min(x1, r.gR) - max(x0, r.gL)); };
        const int64_t ncore = within(r.a0, r.a1) + within(r.b0, r.b1) + within(r.c0, r.c1) + within(r.d0, r.d1);
        if (ncore) atomicAdd(&st->pairs_node_core, (unsigned long long)ncore);
        atomicAdd(&st->pairs_node, (unsigned long long)tot);
        atomicAdd(&st->bins_node, (unsigned long long)tot * (unsigned long long)(min(p.N, w0 + W) - w0));
    }
}

// Per level-0 tile [w0, w1): candidate lines and their split into edge / node-handled / far / mid / centre ranges.
// A line is "interior" for the tile when every bin of the tile lies inside its extent and at
// |t| >= max(2 KB, sqrt(Z) a): then |z|^2 >= Z for every (line, bin) pair (Z = Z1: far, Z = Z2: mid)
// and the interior kernels may run mask-free.  alpha_D = beta nu0 is a function of the centre, so the
// condition is a bound on the centre bin alone; all bounds are conservative.
__global__ void __launch_bounds__(256) range_kernel(Params p, Levels lv, const int32_t* __restrict__ keys, int32_t n,
                                                    TileRange* __restrict__ tr, int32_t* __restrict__ cnt_far,
                                                    int32_t* __restrict__ cnt_mid, int32_t* __restrict__ cnt_edge,
                                                    int32_t* __restrict__ cnt_centre, int32_t* __restrict__ cnt_near,
                                                    int32_t* __restrict__ cnt_lane, DevStats* __restrict__ st)
{
    int wt = blockIdx.x * blockDim.x + threadIdx.x;
    if (wt >= p.n_ct) return;
    apply_shift_bound(p, st);
    const int wb = 32 * p.kb;
    const int64_t mind = (int64_t)kMinDistPerKB * p.kb;
    const int64_t w0 = (int64_t)wt * wb;
    const int64_t w1 = min(p.N, w0 + wb);
    const int32_t n_act = lower_bound_key(keys, n, (int64_t)p.ksent);
    int64_t jlo, jhi;                       // candidate centre bins
    if (p.uncut) { jlo = -kBigKey; jhi = kBigKey; }
    else { jlo = w0 - p.cb_ceil - 2; jhi = w1 - 1 + p.cb_ceil + 2; }
    TileRange r;
    r.A0 = idx_of(p, keys, n_act, jlo);
    r.A1 = idx_of(p, keys, n_act, jhi + 1);
    // left of the tile: the extent must reach the tile's last bin (jc >= jLmin)
    const int64_t jLmin = p.uncut ? -kBigKey : w1 - p.cb_floor;
    int64_t jLfar = min(left_bound((double)w0, p.kappa1, p.inv1p_k1, p.numin_bins), w0 - 1 - mind);
    int64_t jLmid = min(left_bound((double)w0, p.kappa2, p.inv1p_k2, p.numin_bins), w0 - 1 - mind);
    // right of the tile: the extent must reach the tile's first bin (jc <= jRmax)
    const int64_t jRmax = p.uncut ? kBigKey : w0 + p.cb_floor - 2;
    int64_t jRfar = max(right_bound((double)(w1 - 1), p.kappa1, p.inv1m_k1, p.numin_bins), w1 - 1 + mind);
    int64_t jRmid = max(right_bound((double)(w1 - 1), p.kappa2, p.inv1m_k2, p.numin_bins), w1 - 1 + mind);
    if (p.mode == 1) { jLfar = jLmid = -kBigKey; jRfar = jRmid = kBigKey; }
    if (p.mode == 2) { jLfar = -kBigKey; jRfar = kBigKey; }
    int32_t fl0 = idx_of(p, keys, n_act, jLmin);
    int32_t fl1 = idx_of(p, keys, n_act, jLfar + 1);
    int32_t ml1 = idx_of(p, keys, n_act, jLmid + 1);
    int32_t mr0 = idx_of(p, keys, n_act, jRmid);
    int32_t fr0 = idx_of(p, keys, n_act, jRfar);
    int32_t fr1 = idx_of(p, keys, n_act, jRmax + 1);
    // make the sequence monotone inside [A0, A1]; every adjustment only shrinks an interior class
    fl0 = min(max(fl0, r.A0), r.A1);
    fl1 = min(max(fl1, fl0), r.A1);
    ml1 = min(max(ml1, fl1), r.A1);
    fr1 = max(min(fr1, r.A1), ml1);
    fr0 = max(min(fr0, fr1), ml1);
    mr0 = max(min(mr0, fr0), ml1);
    // formula-uniform parts of the edge and centre segments (the rest stays with the generic near kernel):
    //   edge, no core : the tile is only partly inside the extent, but |z|^2 >= Z2 on all of it
    //   centre, full  : the tile is inside the extent; bins with |z|^2 < Z2 exist
    r.EL = r.A0; r.ER = r.A1; r.CL = ml1; r.CR = ml1;
    if (p.mode == 0 || p.mode == 3) {
        r.EL = min(max(idx_of(p, keys, n_act, jLmid + 1), r.A0), fl0);
        r.ER = max(min(idx_of(p, keys, n_act, jRmid), r.A1), fr1);
        r.CL = min(max(idx_of(p, keys, n_act, jLmin), ml1), mr0);
        r.CR = min(max(idx_of(p, keys, n_act, jRmax + 1), r.CL), mr0);
    }
    // node-handled lines (this tile's nodes or an ancestor's): a prefix of the left interior classes and a
    // suffix of the right ones.  With core_nodes the prefix / suffix may reach into the centre class [CL, CR) (separated
    // tiles of the core outside the inner region): every class in between gives way
    int32_t nl = fl0, nrr = fr1;
    if (lv.n_levels > 0) {
        const NodeKeys k = node_keys(p, w0, wb);
        const bool core = p.core_nodes && p.mode == 0;
        nl = min(max(idx_of(p, keys, n_act, k.upL + 1), fl0), core ? r.CR : ml1);
        nrr = max(min(idx_of(p, keys, n_act, k.dnR), fr1), core ? max(r.CL, nl) : mr0);
    }
    fl1 = max(fl1, nl);
    fr0 = min(fr0, nrr);
    ml1 = max(ml1, nl);  r.CL = max(r.CL, nl);       // (no-ops unless core_nodes)
    mr0 = min(mr0, nrr); r.CR = max(min(r.CR, nrr), r.CL);
    r.FL0 = fl0; r.NL = nl; r.FL1 = fl1; r.ML1 = ml1; r.MR0 = mr0; r.FR0 = fr0; r.NR = nrr; r.FR1 = fr1;
    // lane-pass candidates (centre_setup, hk_centre.cuh): innermost bins lie within sqrt(ZG) alpha_D of the centre
    // (z3_for <= HK_ZG; the binned Gaussian: 1/2 + 6 alpha_D), or within the whole core of a line narrower than
    // 0.224 kb/2 bins (25 alpha_D < 5.6 kb/2 bins); centre_setup's own test is 0.2 % generous, kappa3 0.5 %
    r.LL = r.CL; r.LR = r.CR;
    if (p.mode == 0 || p.mode == 3) {
        const int64_t dmin = 6 * (int64_t)(p.kb / 2) + 3;
        double kap3 = p.kappa3, i1p = p.inv1p_k3, i1m = p.inv1m_k3;
        if (p.lane_tight) {
            // the largest z3_for(y^2) over this launch's lines (line_record): 30.25 for a list with y^2 >= 1e-6 throughout
            const float z3m = __uint_as_float((unsigned)st->z3max_bits);
            if (z3m > 0.f && z3m < HK_ZG) { kap3 = sqrt((double)z3m) * p.beta * 1.005; i1p = 1.0 / (1.0 + kap3); i1m = 1.0 / (1.0 - kap3); }
        }
        const int64_t jLl = min(left_bound((double)w0, kap3, i1p, p.numin_bins), w0 - 1 - dmin);
        const int64_t jRl = max(right_bound((double)(w1 - 1), kap3, i1m, p.numin_bins), w1 - 1 + dmin);
        r.LL = min(max(idx_of(p, keys, n_act, jLl + 1), r.CL), r.CR);
        r.LR = max(min(idx_of(p, keys, n_act, jRl), r.CR), r.LL);
    }
    if (p.edge_nodes && p.mode == 0 && lv.n_levels > 0 && !p.uncut) {
        // [A0, ESL) and [ESR, A1) go to edge_node_kernel; the direct edge kernel keeps [ESL, EL) and [ER, ESR)
        const EdgeKeys ek = edge_keys(p, w0, wb);
        r.A0 = min(max(idx_of(p, keys, n_act, ek.upL + 1), r.A0), r.EL);
        r.A1 = max(min(idx_of(p, keys, n_act, ek.dnR), r.A1), r.ER);
    }
    tr[wt] = r;
    const unsigned long long nb = (unsigned long long)(w1 - w0);
    const long long nfar = (long long)(fl1 - nl) + (nrr - fr0);
    const long long nmid = (long long)(ml1 - fl1) + (fr0 - mr0);
    const long long nedge = (long long)(r.EL - r.A0) + (r.A1 - r.ER);
    const long long ncen = (long long)(r.CR - r.CL);
    const long long nnear = (long long)(fl0 - r.EL) + (r.CL - ml1) + (mr0 - r.CR) + (r.ER - fr1);
    cnt_far[wt] = (int32_t)((nfar + p.chunk - 1) / p.chunk);
    cnt_mid[wt] = (int32_t)((nmid + p.chunk - 1) / p.chunk);
    cnt_edge[wt] = (int32_t)((nedge + p.chunk - 1) / p.chunk);
    cnt_centre[wt] = (int32_t)((ncen + p.chunk_centre - 1) / p.chunk_centre);
    cnt_lane[wt] = (int32_t)(((long long)(r.LR - r.LL) + p.chunk_lane - 1) / p.chunk_lane);
    cnt_near[wt] = (int32_t)((nnear + p.chunk - 1) / p.chunk);
    if (nfar) atomicAdd(&st->pairs_far, (unsigned long long)nfar * nb);
    if (nmid) atomicAdd(&st->pairs_mid, (unsigned long long)nmid * nb);
    if (nedge) atomicAdd(&st->pairs_edge, (unsigned long long)nedge * nb);
    if (ncen) atomicAdd(&st->pairs_centre, (unsigned long long)ncen * nb);
    if (nnear) atomicAdd(&st->pairs_near, (unsigned long long)nnear * nb);
}

}  // namespace hk
