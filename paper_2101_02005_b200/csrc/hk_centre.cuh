// hk_centre.cuh -- step a4 of the hot path: the line centres.  Two kernels over the same work units
// (a level-0 tile inside the extent x a chunk of the sorted lines whose centre lies within two tiles of it or whose
// core reaches it -- TileRange [CL, CR)):
//
//   centre_row_kernel<KB>        lanes own bins, the warp walks lines.  Every (line, tile) visit is ONE packed rational
//        function of X = ((nu_i - nu0)/alpha_D)^2 whose coefficients depend on the line only: they are worked out once
//        per visit by the lane that stages the line (32 lines at a time, one per lane) and read back as broadcast
//        shared-memory loads, so a visit costs two Horner chains, one reciprocal and no branch.  Visits are bucketed
//        by formula when they are staged and each bucket runs its own tight loop:
//            R2   two asymptotic terms                  (every bin of the tile has |z|^2 >= Z2)
//            R4   4-point Gauss-Hermite, cubic/quartic  (every bin has |z|^2 >= Z4)
//            R6m  6-point Gauss-Hermite, quintic/sextic (the tile holds bins with |z|^2 < Z4), zero where X < xl
//            R10  10-point Gauss-Hermite, degree 9/10   (the tile holds bins with |z|^2 < Z3 of a line with y >= 1.8)
//            R2m  two terms, zero where X < xl          (lines narrower than a fifth of a bin: the whole core is lane work)
//        A warp is a work unit of its own (no block-level synchronisation anywhere); its 32 KB bins reach k(nu) with one
//        fp64 atomic per bin per unit.
//   centre_lane_kernel<KB,W,kBinned>   the innermost bins, X < xl (|z| < 5.5, or the whole core of a narrow line):
//        lane <-> line, 32 lines step through the same bins, each evaluating its own line there -- 10-point
//        Gauss-Hermite (y >= 1.8), trapezoid rule with pole term (y < 1.8), the bare Gaussian (y = 0) or the bin-averaged
//        Gaussian.  A batch is counting-sorted by y = Gamma_L/alpha_D when it is staged, so the 32 lines of a group
//        share evaluator and ring width.  Values go through a shared staging matrix and are summed per bin (a
//        transpose, no atomics).
//
// Both kernels decide "row or lane" for a bin from the SAME fp32 operations on the same record (centre_setup, X below),
// so every bin of every visit is evaluated exactly once.
//
// The Gauss-Hermite forms: K = (y/pi) sum_k w_k/((x - t_k)^2 + y^2); the node pairs +-t_k combine to
//   K = y sum_k W_k (X + c_k)/D_k(X),  D_k = X^2 + 2 (y^2 - T_k) X + c_k^2,  c_k = y^2 + T_k, T_k = t_k^2, W_k = 2 w_k/pi,
// a rational function N(X)/D(X) of X = x^2 with D = prod D_k monic (what the paper's regions A and B do with 1 and 3
// nodes, Table 1).  Measured against the oracle (tests/test_gpu_parity.py::test_evaluator_accuracy_map):
// 4 points <= 1.0e-6 for |z| >= 8, 6 points <= 7.7e-6 for |z| >= 5.5.
#pragma once
#include "hk_gh_tables.cuh"

namespace hk {

constexpr int kRowNone = 0, kRowR2 = 1, kRowR2m = 2, kRowR4 = 3, kRowR6m = 4, kRowR10 = 5;
constexpr int kLaneNone = 0, kLaneGH10 = 1, kLaneTrap = 2, kLaneGauss = 3, kLaneFull = 4, kLaneBinned = 5;

struct CentreLine {
    int row, lane;          // row class of this (line, tile) visit; evaluator of its lane-pass bins (none: no such bins)
    float ndl, nf;          // -(jp - tile start), -f: t = (b + ndl) + nf
    float inva, nfa;        // dnu/alpha_D (0 for the Lorentz profile) and -f inva: u = fma(b + ndl, inva, nfa), X = u u
    float xl;               // rows take the bins with X >= xl, the lane pass those with X < xl
    float y2, G2, c, ip, flo;
};

// Everything both kernels need to know about one (line, tile) visit.  ra = recA = { jp, f, G2 | flo, c },
// rc = recC = { inva, nfa, y2, ip }: the per-line part (IEEE square roots and divisions, once per line, gather_kernel).
template <int KB>
__device__ __forceinline__ CentreLine centre_setup(const float4 ra, const float4 rc, const int64_t ct0, const int profile)
{
    constexpr float whi = (float)(32 * KB - 1);
    CentreLine L;
    // (32-bit difference: a line of this tile's centre range lies within a core radius of the tile)
    const float fdj = (float)(__float_as_int(ra.x) - (int)ct0);
    const bool binned = profile == HK_PROFILE_BINNED_GAUSSIAN;
    L.ndl = -fdj; L.nf = -ra.y;
    L.G2 = binned ? 0.f : ra.z; L.flo = binned ? ra.z : 0.f;         // (binned: the slot carries the low part of f)
    L.c = ra.w;
    L.inva = rc.x; L.nfa = rc.y; L.y2 = rc.z; L.ip = rc.w;
    L.row = L.c != 0.f ? kRowR2 : kRowNone;
    L.lane = kLaneNone; L.xl = -1.0f;
    if (!(L.inva > 0.f)) return L;               // Lorentz profile: every formula is the exact Lorentzian, no core
    // smallest X over the tile's bins, from below
    const float pos = fdj + ra.y;
    const float umin = fmaxf(fmaxf(-pos, pos - whi), 0.f) * 0.999f * L.inva;
    const float Xmin = umin * umin * 0.999f;
    if (binned) {
        const float h = fmaf(0.5f, L.inva, 6.0f);                      // |t| < 1/2 + 6 a
        L.xl = h * h;
        L.row = kRowNone;
        L.lane = Xmin < L.xl ? kLaneBinned : kLaneNone;
        return L;
    }
    if (L.y2 >= HK_Z2) return L;                 // |z|^2 >= Z2 everywhere
    // (ip = 0: G = 0, the pure Gaussian, whose row formulas are all zero -- or an amplitude below the launch's range)
    const bool has_gh = L.ip > 0.f;
    // narrower than about a fifth of a bin per 64 bins of tile: X would leave the range the expanded polynomials are
    // good for, and the core spans a handful of bins -- two-term rows, the whole core in the lane pass
    constexpr float kNarrow = 4.4721360f / (float)(KB / 2);             // 1/inva < sqrt(0.05) KB/2
    if (L.inva > kNarrow) {
        const float xc = HK_Z2 - L.y2;
        if (Xmin < xc) {
            L.xl = xc;
            L.row = L.c != 0.f ? kRowR2m : kRowNone;
            L.lane = L.y2 == 0.f ? kLaneGauss : kLaneFull;
        }
        return L;
    }
    if (Xmin + L.y2 >= HK_Z2) return L;          // no core bin in this tile
    const float z3 = z3_for(L.y2);                                 // (both shrink to nothing as y grows: hk_device.cuh)
    if (Xmin + L.y2 >= fmaxf(z4_for(L.y2), z3)) { L.row = has_gh ? kRowR4 : kRowNone; return L; }
    L.xl = z3 - L.y2;                                              // (<= 0 for y >= 3: the 6-point rows take the whole tile)
    L.row = has_gh ? kRowR6m : kRowNone;
    if (L.xl > 0.f && Xmin < L.xl) {
        // innermost bins.  y >= 1.8 (HK_Y10): the 10-point rule converges on all of them -- as a row over the whole tile when X^10
        // stays inside fp32 (a >= 0.85 bins per 64 bins of tile), else in the lane pass.  y < 1.8: trapezoid rule, lane pass
        constexpr float kWide = 1.0f / (0.85f * (float)(KB / 2));
        if (L.y2 >= HK_Y10 * HK_Y10 && has_gh && L.inva < kWide) { L.row = kRowR10; L.xl = -1.0f; }
        else L.lane = L.y2 == 0.f ? kLaneGauss : L.y2 >= HK_Y10 * HK_Y10 ? kLaneGH10 : kLaneTrap;
    }
    return L;
}

// ---- coefficients of the expanded Gauss-Hermite forms: polynomials in Y = y^2 (hk_gh_tables.cuh) -------------------
template <int NC>
__device__ __forceinline__ float horner_y(const float (&c)[NC], float Y)
{
    float v = c[0];
#pragma unroll
    for (int i = 1; i < NC; ++i) v = fmaf(v, Y, c[i]);
    return v;
}
constexpr float kGhN = 0.5641895835477563f;      // leading coefficient of every N: sum_k W_k = 1/sqrt(pi)

// 4 points: K/y = (kGhN X^3 + n[2] X^2 + n[1] X + n[0]) / (X^4 + d[3] X^3 + d[2] X^2 + d[1] X + d[0])
__device__ __forceinline__ void gh4_coeffs(float Y, float (&n)[3], float (&d)[4])
{
    n[0] = horner_y(kGh4N0, Y); n[1] = horner_y(kGh4N1, Y); n[2] = horner_y(kGh4N2, Y);
    d[0] = horner_y(kGh4D0, Y); d[1] = horner_y(kGh4D1, Y); d[2] = horner_y(kGh4D2, Y); d[3] = horner_y(kGh4D3, Y);
}
// 6 points: K/y = (kGhN X^5 + n[4] X^4 + ... + n[0]) / (X^6 + d[5] X^5 + ... + d[0])
__device__ __forceinline__ void gh6_coeffs(float Y, float (&n)[5], float (&d)[6])
{
    n[0] = horner_y(kGh6N0, Y); n[1] = horner_y(kGh6N1, Y); n[2] = horner_y(kGh6N2, Y); n[3] = horner_y(kGh6N3, Y);
    n[4] = horner_y(kGh6N4, Y);
    d[0] = horner_y(kGh6D0, Y); d[1] = horner_y(kGh6D1, Y); d[2] = horner_y(kGh6D2, Y); d[3] = horner_y(kGh6D3, Y);
    d[4] = horner_y(kGh6D4, Y); d[5] = horner_y(kGh6D5, Y);
}
// 10 points: K/y = (kGhN X^9 + n[8] X^8 + ... + n[0]) / (X^10 + d[9] X^9 + ... + d[0])
__device__ __forceinline__ void gh10_coeffs(float Y, float (&n)[9], float (&d)[10])
{
    n[0] = horner_y(kGh10N0, Y); n[1] = horner_y(kGh10N1, Y); n[2] = horner_y(kGh10N2, Y); n[3] = horner_y(kGh10N3, Y);
    n[4] = horner_y(kGh10N4, Y); n[5] = horner_y(kGh10N5, Y); n[6] = horner_y(kGh10N6, Y); n[7] = horner_y(kGh10N7, Y);
    n[8] = horner_y(kGh10N8, Y);
    d[0] = horner_y(kGh10D0, Y); d[1] = horner_y(kGh10D1, Y); d[2] = horner_y(kGh10D2, Y); d[3] = horner_y(kGh10D3, Y);
    d[4] = horner_y(kGh10D4, Y); d[5] = horner_y(kGh10D5, Y); d[6] = horner_y(kGh10D6, Y); d[7] = horner_y(kGh10D7, Y);
    d[8] = horner_y(kGh10D8, Y); d[9] = horner_y(kGh10D9, Y);
}
// the same forms for one evaluation (accuracy probe): Re w(x + i y) with X = x^2, Y = y^2
__device__ __forceinline__ float gh10_row_K(float X, float Y, float y)
{
    float n[9], d[10];
    gh10_coeffs(Y, n, d);
    float N = kGhN, D = X + d[9];
#pragma unroll
    for (int i = 8; i >= 0; --i) { N = fmaf(N, X, n[i]); D = fmaf(D, X, d[i]); }
    return y * N * rcp_approx(D);
}
__device__ __forceinline__ float gh4_row_K(float X, float Y, float y)
{
    float n[3], d[4];
    gh4_coeffs(Y, n, d);
    const float N = fmaf(fmaf(fmaf(kGhN, X, n[2]), X, n[1]), X, n[0]);
    const float D = fmaf(fmaf(fmaf(X + d[3], X, d[2]), X, d[1]), X, d[0]);
    return y * N * rcp_approx(D);
}
__device__ __forceinline__ float gh6_row_K(float X, float Y, float y)
{
    float n[5], d[6];
    gh6_coeffs(Y, n, d);
    const float N = fmaf(fmaf(fmaf(fmaf(fmaf(kGhN, X, n[4]), X, n[3]), X, n[2]), X, n[1]), X, n[0]);
    const float D = fmaf(fmaf(fmaf(fmaf(fmaf(X + d[5], X, d[4]), X, d[3]), X, d[2]), X, d[1]), X, d[0]);
    return y * N * rcp_approx(D);
}

// ---------------------------------------------------------------------------------------
// row kernel
// ---------------------------------------------------------------------------------------
constexpr int kRowWarps = 8;           // warps per CTA (independent of each other)
constexpr int kRowCtas = 4;            // resident CTAs per SM the kernel is compiled and launched for

template <int KB>
__global__ void __launch_bounds__(32 * kRowWarps, kRowCtas) centre_row_kernel(AccArgs a)
{
    constexpr int M = KB / 2;
    constexpr int kTB = 32 * KB;
    // per warp: the row records of the 32 staged lines, bucketed by class.  float4 x 4 per record:
    //   R2 / R2m: A = { ndl, nf, G2, c },       B = { 1.5 a^2, -2 a^2 G^2, inva, nfa },  C = { xl, ... }
    //   R4      : A = { -, u0 = ndl inva + nfa, inva, 1/P },  B = { n0, n1, n2, d3/P },  C = { d0/P, d1/P, d2/P, - }
    //   R6m     : A = { ndl, nfa, inva, xl },   B = { n0, n1, n2, n3 },  C = { n4, d0/P, d1/P, d2/P },  D = { d3/P, d4/P, d5/P, 1/P }
    //   R10     : A = { ndl, nfa, inva, 1/P },  B, C = { n0 .. n7 },  D = { n8, d0/P, d1/P, d2/P },  E = { d3/P .. d6/P },  F = { d7/P, d8/P, d9/P, - }
    //   (P = cK y, the amplitude of the Gauss-Hermite forms, divides the DENOMINATOR's coefficients: the leading 1 becomes
    //    1/P at no cost, the numerator stays in range for any amplitude, and a denominator that overflows -- a line 40
    //    orders of magnitude below the strongest -- gives a reciprocal of zero)
    __shared__ float4 rec[kRowWarps][6][32];
    // Visits of the two heavy classes (R6m, R10) are not expanded where they are staged -- that would run ~130 divergent
    // instructions per batch for the few lanes that need them -- but PARKED ({ ndl, nfa, inva, xl | ip }, { y^2, ip }),
    // and expanded 32 at a time, every lane busy on the same polynomial tables, when a park fills up or the unit ends.
    __shared__ float4 park[kRowWarps][2][2][32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    float4 (*rw)[32] = rec[warp];
    float4 (*pk6)[32] = park[warp][0];
    float4 (*pk10)[32] = park[warp][1];
    const int32_t* __restrict__ prefix = a.prefix_centre;
    const int base = prefix[0], total = prefix[a.n_ct];
    const unsigned lt_mask = (1u << lane) - 1u;

    float2 tb[M];
#pragma unroll
    for (int m = 0; m < M; ++m) {
        float b0 = (float)(lane + 64 * m);
        tb[m] = make_float2(b0, b0 + 32.0f);
    }

    for (;;) {
        int u = 0;
        if (lane == 0) u = (int)atomicAdd(&a.st->unit_counter_centre, 1u);
        u = __shfl_sync(0xffffffffu, u, 0) + base;
        if (u >= total) break;
        const int ct = find_tile(prefix, a.n_ct, u);
        const int64_t ct0 = (int64_t)ct * kTB;
        const int c0 = a.tr[ct].CL + (u - prefix[ct]) * a.chunk_centre;
        const int nt = min(a.chunk_centre, a.tr[ct].CR - c0);
        if (nt <= 0) continue;
        if (lane == 0) atomicAdd(&a.st->units_centre, 1ULL);

        float2 acc[M];
        double acc64[KB];
#pragma unroll
        for (int m = 0; m < M; ++m) acc[m] = make_float2(0.f, 0.f);
#pragma unroll
        for (int j = 0; j < KB; ++j) acc64[j] = 0.0;
        int since = 0;                          // lines whose terms the fp32 partial sums hold (at most kFlush + 64)
        auto spill = [&]() {
            if (since >= kFlush - 32) {
#pragma unroll
                for (int m = 0; m < M; ++m) {
                    acc64[2 * m] += (double)acc[m].x;
                    acc64[2 * m + 1] += (double)acc[m].y;
                    acc[m] = make_float2(0.f, 0.f);
                }
                since = 0;
            }
        };
        // ---- R6m: P N(X)/D(X), quintic over monic sextic, zero where X < xl; records rw[0..3][0..n)
        auto run_r6 = [&](int n) {
#pragma unroll 2
            for (int l = 0; l < n; ++l) {
                const float4 ea = rw[0][l], eb = rw[1][l], ec = rw[2][l], ed = rw[3][l];
                const float2 ndl = bcast2(ea.x), nfa = bcast2(ea.y), ia = bcast2(ea.z);
                const float xl = ea.w;
                const float2 n0 = bcast2(eb.x), n1 = bcast2(eb.y), n2c = bcast2(eb.z), n3 = bcast2(eb.w);
                const float2 n4c = bcast2(ec.x), d0 = bcast2(ec.y), d1 = bcast2(ec.z), d2 = bcast2(ec.w);
                const float2 d3 = bcast2(ed.x), d4 = bcast2(ed.y), d5 = bcast2(ed.z), ip = bcast2(ed.w), n5 = bcast2(kGhN);
#pragma unroll
                for (int m = 0; m < M; ++m) {
                    const float2 d = __fadd2_rn(tb[m], ndl);
                    const float2 un = __ffma2_rn(d, ia, nfa);
                    const float2 X = __fmul2_rn(un, un);
                    float2 N = __ffma2_rn(n5, X, n4c);
                    N = __ffma2_rn(N, X, n3);
                    N = __ffma2_rn(N, X, n2c);
                    N = __ffma2_rn(N, X, n1);
                    N = __ffma2_rn(N, X, n0);
                    float2 Dn = __ffma2_rn(X, ip, d5);
                    Dn = __ffma2_rn(Dn, X, d4);
                    Dn = __ffma2_rn(Dn, X, d3);
                    Dn = __ffma2_rn(Dn, X, d2);
                    Dn = __ffma2_rn(Dn, X, d1);
                    Dn = __ffma2_rn(Dn, X, d0);
                    float2 R = rcp2(Dn);
                    R.x = X.x >= xl ? R.x : 0.f;                        // the lane pass owns these bins
                    R.y = X.y >= xl ? R.y : 0.f;
                    acc[m] = __ffma2_rn(N, R, acc[m]);
                }
            }
        };
        // ---- R10: N(X)/D'(X), degree 9 over degree 10, the whole tile (y >= 1.8); records rw[0..5][0..n)
        auto run_r10 = [&](int n) {
#pragma unroll 1
            for (int l = 0; l < n; ++l) {
                const float4 ea = rw[0][l], eb = rw[1][l], ec = rw[2][l], ed = rw[3][l], ee = rw[4][l], ef = rw[5][l];
                const float2 ndl = bcast2(ea.x), nfa = bcast2(ea.y), ia = bcast2(ea.z), ip = bcast2(ea.w);
#pragma unroll
                for (int m = 0; m < M; ++m) {
                    const float2 d = __fadd2_rn(tb[m], ndl);
                    const float2 un = __ffma2_rn(d, ia, nfa);
                    const float2 X = __fmul2_rn(un, un);
                    float2 N = __ffma2_rn(bcast2(kGhN), X, bcast2(ed.x));
                    N = __ffma2_rn(N, X, bcast2(ec.w));
                    N = __ffma2_rn(N, X, bcast2(ec.z));
                    N = __ffma2_rn(N, X, bcast2(ec.y));
                    N = __ffma2_rn(N, X, bcast2(ec.x));
                    N = __ffma2_rn(N, X, bcast2(eb.w));
                    N = __ffma2_rn(N, X, bcast2(eb.z));
                    N = __ffma2_rn(N, X, bcast2(eb.y));
                    N = __ffma2_rn(N, X, bcast2(eb.x));
                    float2 Dn = __ffma2_rn(X, ip, bcast2(ef.z));
                    Dn = __ffma2_rn(Dn, X, bcast2(ef.y));
                    Dn = __ffma2_rn(Dn, X, bcast2(ef.x));
                    Dn = __ffma2_rn(Dn, X, bcast2(ee.w));
                    Dn = __ffma2_rn(Dn, X, bcast2(ee.z));
                    Dn = __ffma2_rn(Dn, X, bcast2(ee.y));
                    Dn = __ffma2_rn(Dn, X, bcast2(ee.x));
                    Dn = __ffma2_rn(Dn, X, bcast2(ed.w));
                    Dn = __ffma2_rn(Dn, X, bcast2(ed.z));
                    Dn = __ffma2_rn(Dn, X, bcast2(ed.y));
                    acc[m] = __ffma2_rn(N, rcp2(Dn), acc[m]);
                }
            }
        };
        int cnt6 = 0, cnt10 = 0;                // parked visits (warp-uniform)
        // expand the parked visits of one class into row records and evaluate them (rw must be free: call after a __syncwarp
        // that follows its last read)
        auto flush6 = [&]() {
            if (lane < cnt6) {
                const float4 p0 = pk6[0][lane], p1 = pk6[1][lane];
                float n[5], d[6];
                gh6_coeffs(p1.x, n, d);
                const float ip = p1.y;
                rw[0][lane] = p0;                                        // { ndl, nfa, inva, xl }
                rw[1][lane] = make_float4(n[0], n[1], n[2], n[3]);
                rw[2][lane] = make_float4(n[4], d[0] * ip, d[1] * ip, d[2] * ip);
                rw[3][lane] = make_float4(d[3] * ip, d[4] * ip, d[5] * ip, ip);
            }
            __syncwarp();
            run_r6(cnt6);
            since += cnt6; cnt6 = 0;
            spill();
            __syncwarp();
        };
        auto flush10 = [&]() {
            if (lane < cnt10) {
                const float4 p0 = pk10[0][lane], p1 = pk10[1][lane];
                float n[9], d[10];
                gh10_coeffs(p1.x, n, d);
                const float ip = p1.y;
                rw[0][lane] = p0;                                        // { ndl, nfa, inva, ip }
                rw[1][lane] = make_float4(n[0], n[1], n[2], n[3]);
                rw[2][lane] = make_float4(n[4], n[5], n[6], n[7]);
                rw[3][lane] = make_float4(n[8], d[0] * ip, d[1] * ip, d[2] * ip);
                rw[4][lane] = make_float4(d[3] * ip, d[4] * ip, d[5] * ip, d[6] * ip);
                rw[5][lane] = make_float4(d[7] * ip, d[8] * ip, d[9] * ip, 0.f);
            }
            __syncwarp();
            run_r10(cnt10);
            since += cnt10; cnt10 = 0;
            spill();
            __syncwarp();
        };

        float4 ra = make_float4(0.f, 0.f, 1.f, 0.f), rcc = make_float4(0.f, 0.f, 0.f, 0.f);
        if (lane < nt) { ra = a.recA[c0 + lane]; rcc = a.recC[c0 + lane]; }
        for (int v0 = 0; v0 < nt; v0 += 32) {
            // ---- stage 32 lines: one per lane
            int rc = kRowNone;
            float4 A, B, C, P1;
            A = B = C = P1 = make_float4(0.f, 0.f, 0.f, 0.f);
            if (v0 + lane < nt) {
                const CentreLine L = centre_setup<KB>(ra, rcc, ct0, a.profile);
                rc = L.row;
                const float ip = L.ip;
                if (rc == kRowR4) {
                    float n[3], d[4];
                    gh4_coeffs(L.y2, n, d);
                    // (u = b inva + u0 with u0 = ndl inva + nfa: no bin of an R4 visit is masked, so its u need not match the
                    //  lane pass bit for bit, and |u0| <= 64 inva ulps are far inside the evaluator's budget)
                    A = make_float4(0.f, __fmaf_rn(L.ndl, L.inva, L.nfa), L.inva, ip);
                    B = make_float4(n[0], n[1], n[2], d[3] * ip);
                    C = make_float4(d[0] * ip, d[1] * ip, d[2] * ip, 0.f);
                } else if (rc == kRowR6m || rc == kRowR10) {
                    A = make_float4(L.ndl, L.nfa, L.inva, rc == kRowR6m ? L.xl : ip);
                    P1 = make_float4(L.y2, ip, 0.f, 0.f);
                } else if (rc == kRowR2 || rc == kRowR2m) {
                    const float a2 = L.inva > 0.f ? rcp_approx(L.inva * L.inva) : 0.f;   // (second-order term only)
                    A = make_float4(L.ndl, L.nf, L.G2, L.c);
                    B = make_float4(1.5f * a2, -2.0f * a2 * L.G2, L.inva, L.nfa);
                    C = make_float4(L.xl, 0.f, 0.f, 0.f);
                }
            }
            // next batch's records: in flight while this one is evaluated
            if (v0 + 32 + lane < nt) { ra = a.recA[c0 + v0 + 32 + lane]; rcc = a.recC[c0 + v0 + 32 + lane]; }
            const unsigned m2 = __ballot_sync(0xffffffffu, rc == kRowR2), m2m = __ballot_sync(0xffffffffu, rc == kRowR2m);
            const unsigned m4 = __ballot_sync(0xffffffffu, rc == kRowR4), m6 = __ballot_sync(0xffffffffu, rc == kRowR6m);
            const unsigned m10 = __ballot_sync(0xffffffffu, rc == kRowR10);
            const int n2 = __popc(m2), n2m = __popc(m2m), n4 = __popc(m4), n6 = __popc(m6), n10 = __popc(m10);
            __syncwarp();                       // the previous batch's records are consumed
            // park the heavy visits (a park that would overflow is worked off first)
            if (cnt6 + n6 > 32) flush6();
            if (cnt10 + n10 > 32) flush10();
            if (rc == kRowR6m) { const int s = cnt6 + __popc(m6 & lt_mask); pk6[0][s] = A; pk6[1][s] = P1; }
            if (rc == kRowR10) { const int s = cnt10 + __popc(m10 & lt_mask); pk10[0][s] = A; pk10[1][s] = P1; }
            cnt6 += n6; cnt10 += n10;
            int slot = -1;
            if (rc == kRowR2) slot = __popc(m2 & lt_mask);
            else if (rc == kRowR2m) slot = n2 + __popc(m2m & lt_mask);
            else if (rc == kRowR4) slot = n2 + n2m + __popc(m4 & lt_mask);
            if (slot >= 0) {
                rw[0][slot] = A; rw[1][slot] = B;
                if (rc >= kRowR2m) rw[2][slot] = C;
            }
            __syncwarp();
            int l = 0;
            // ---- R2: c r (1 + r (A1 - A2 r)), r = 1/(t^2 + G^2)
#pragma unroll 4
            for (; l < n2; ++l) {
                const float4 ea = rw[0][l];
                const float2 eb = *reinterpret_cast<const float2*>(&rw[1][l]);
                const float2 ndl = bcast2(ea.x), nf = bcast2(ea.y), g = bcast2(ea.z), c = bcast2(ea.w);
                const float2 A1 = bcast2(eb.x), nA2 = bcast2(eb.y), one = bcast2(1.0f);
#pragma unroll
                for (int m = 0; m < M; ++m) {
                    const float2 d = __fadd2_rn(tb[m], ndl);          // exact: both are small integers
                    const float2 t = __fadd2_rn(d, nf);
                    const float2 q = __ffma2_rn(t, t, g);
                    const float2 rr = rcp2(q);
                    const float2 uu = __ffma2_rn(nA2, rr, A1);
                    const float2 vv = __ffma2_rn(uu, rr, one);
                    acc[m] = __ffma2_rn(c, __fmul2_rn(rr, vv), acc[m]);
                }
            }
            // ---- R2m: the same, zero where X < xl
            const int e2m = n2 + n2m;
#pragma unroll 1
            for (; l < e2m; ++l) {
                const float4 ea = rw[0][l], eb = rw[1][l];
                const float2 ndl = bcast2(ea.x), nf = bcast2(ea.y), g = bcast2(ea.z), c = bcast2(ea.w);
                const float2 A1 = bcast2(eb.x), nA2 = bcast2(eb.y), one = bcast2(1.0f), ia = bcast2(eb.z), nfa = bcast2(eb.w);
                const float xl = rw[2][l].x;
#pragma unroll
                for (int m = 0; m < M; ++m) {
                    const float2 d = __fadd2_rn(tb[m], ndl);
                    const float2 t = __fadd2_rn(d, nf);
                    const float2 q = __ffma2_rn(t, t, g);
                    const float2 rr = rcp2(q);
                    const float2 uu = __ffma2_rn(nA2, rr, A1);
                    const float2 vv = __ffma2_rn(uu, rr, one);
                    float2 ww = __fmul2_rn(rr, vv);
                    const float2 un = __ffma2_rn(d, ia, nfa);
                    const float2 X = __fmul2_rn(un, un);
                    ww.x = X.x >= xl ? ww.x : 0.f;                      // the lane pass owns these bins
                    ww.y = X.y >= xl ? ww.y : 0.f;
                    acc[m] = __ffma2_rn(c, ww, acc[m]);
                }
            }
            // ---- R4: P N(X)/D(X), cubic over monic quartic
            const int e4 = e2m + n4;
#pragma unroll 4
            for (; l < e4; ++l) {
                const float4 ea = rw[0][l], eb = rw[1][l], ec = rw[2][l];
                const float2 u0 = bcast2(ea.y), ia = bcast2(ea.z), ip = bcast2(ea.w);
                const float2 n0 = bcast2(eb.x), n1 = bcast2(eb.y), n2c = bcast2(eb.z), d3 = bcast2(eb.w);
                const float2 d0 = bcast2(ec.x), d1 = bcast2(ec.y), d2 = bcast2(ec.z), n3 = bcast2(kGhN);
#pragma unroll
                for (int m = 0; m < M; ++m) {
                    const float2 un = __ffma2_rn(tb[m], ia, u0);
                    const float2 X = __fmul2_rn(un, un);
                    float2 N = __ffma2_rn(n3, X, n2c);
                    N = __ffma2_rn(N, X, n1);
                    N = __ffma2_rn(N, X, n0);
                    float2 Dn = __ffma2_rn(X, ip, d3);
                    Dn = __ffma2_rn(Dn, X, d2);
                    Dn = __ffma2_rn(Dn, X, d1);
                    Dn = __ffma2_rn(Dn, X, d0);
                    acc[m] = __ffma2_rn(N, rcp2(Dn), acc[m]);
                }
            }
            // fp32 partial sums hold at most kFlush + 64 lines' terms
            since += e4;
            spill();
        }
        __syncwarp();
        if (cnt6 > 0) flush6();
        if (cnt10 > 0) flush10();
        const double sc = scalbn(1.0, -a.st->scale_exp);
#pragma unroll
        for (int m = 0; m < M; ++m) {
            const double v0 = (acc64[2 * m] + (double)acc[m].x) * sc, v1 = (acc64[2 * m + 1] + (double)acc[m].y) * sc;
            const int64_t b = ct0 + lane + 64 * m;
            if (b < a.N && v0 != 0.0) atomicAdd(a.out_k + b, v0);
            if (b + 32 < a.N && v1 != 0.0) atomicAdd(a.out_k + b + 32, v1);
        }
    }
}

// ---------------------------------------------------------------------------------------
// lane kernel
// ---------------------------------------------------------------------------------------
constexpr int kStage = 16;             // bins per staging step
constexpr int kLaneCtas = 4;           // resident CTAs per SM (8 warps each) the lane kernel is compiled and launched for
constexpr int kYClasses = 32;          // classes the pooled lines are sorted into (one per evaluator: kLane*)

// the value of one (line, bin) pair of the lane pass, amplitude included
__device__ __forceinline__ float lane_value(int type, float cK, float x, float X, float y, float y2, const TrapLine& TL,
                                            const float* __restrict__ wtab)
{
    if (type == kLaneTrap) return cK * trap_K<true>(x, TL, wtab);
    if (type == kLaneGH10) return cK * gh10_K(X, X + y2, y);
    if (type == kLaneGauss) return gauss_term(cK, x);
    return cK * core_any_K(x, y, nullptr);           // narrow lines: every ring of the core
}

// W = warps per CTA: 8 for dense lists; 2 or 1 for sparse ones (few lines per tile: a work unit is a handful of lines,
// and more small CTAs keep more units in flight).
// Only a minority of the (line, tile) visits of a unit has lane-pass bins, so the visits that do are POOLED in shared
// memory across the staged batches; when the pool is full (or the unit ends) it is counting-sorted by evaluator and dealt
// to the warps in groups of 32 -- every warp busy, every lane of a group live and running the same code.  Within a class
// the lines keep (roughly) their order by centre, so the 32 rings of a group overlap and the lanes are busy on the same bins.
template <int KB, int W, bool kBinned>
__global__ void __launch_bounds__(32 * W, (kLaneCtas * 8) / W) centre_lane_kernel(AccArgs a)
{
    constexpr int kWarps = W, kThreads = 32 * W, kSubC = 64 * W, kLPTC = kSubC / kThreads;
    constexpr int kCap = (KB == 8 ? 80 : 96) * W, kPPT = (kCap + kThreads - 1) / kThreads;   // pool capacity; entries per thread
    constexpr int kTB = 32 * KB;
    static_assert(sizeof(double) * kWarps * kTB <= sizeof(float) * kWarps * kStage * 33, "red must fit in the staging matrix");
    __shared__ float4 poolA[kCap];             // { dl, f, inva, xl }
    __shared__ float4 poolB[kCap];             // { cK, y2 | flo, type, - }
    __shared__ unsigned short order[kCap];     // pool indices sorted by y class
    __shared__ __align__(16) float stage[kWarps][kStage][33];
    __shared__ float sacc[kWarps][kTB];
    __shared__ int hist[kYClasses];
    __shared__ int s_unit, s_pool_n, s_next;
    __shared__ __align__(16) float wtab[24];   // trapezoid weights of the two node sets (trap_K)
    trap_weights_to_shared(wtab, threadIdx.x);
    if (kThreads < 24 && threadIdx.x == 0) { for (int i = kThreads; i < 24; ++i) trap_weights_to_shared(wtab, i); }
    const float* const wsh = trap_weights_address(wtab);
    double* red = reinterpret_cast<double*>(&stage[0][0][0]);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int32_t* __restrict__ prefix = a.prefix_lane;
    const int base = prefix[0], total = prefix[a.n_ct];
    const float whi = (float)(kTB - 1);
#pragma unroll
    for (int j = 0; j < KB; ++j) sacc[warp][lane + 32 * j] = 0.f;

    for (;;) {
        const int u = next_unit(&a.st->unit_counter_lane, &s_unit) + base;
        if (u >= total) break;
        const int ct = find_tile(prefix, a.n_ct, u);
        const int64_t ct0 = (int64_t)ct * kTB;
        const TileRange r = a.tr[ct];
        const int c0 = r.LL + (u - prefix[ct]) * a.chunk_lane;       // (lines that can have innermost bins here: range_kernel)
        const int nt = min(a.chunk_lane, r.LR - c0);
        if (nt <= 0) continue;

        double acc64[KB];
#pragma unroll
        for (int j = 0; j < KB; ++j) acc64[j] = 0.0;
        int since_flush = 0;
        bool any_work = false;
        auto flush = [&]() {
            __syncwarp();
#pragma unroll
            for (int j = 0; j < KB; ++j) {
                acc64[j] += (double)sacc[warp][lane + 32 * j];
                sacc[warp][lane + 32 * j] = 0.f;
            }
            since_flush = 0;
            __syncwarp();
        };

        float4 preA[kLPTC], preC[kLPTC];
        float preK[kLPTC];
        auto fetch = [&](int v0) {
#pragma unroll
            for (int k = 0; k < kLPTC; ++k) {
                const int v = v0 + threadIdx.x + k * kThreads;
                if (v < nt) { preA[k] = a.recA[c0 + v]; preC[k] = a.recC[c0 + v]; preK[k] = a.recB[c0 + v].w; }
            }
        };
        // one group of up to 32 pooled lines: the lanes step through the same bins, each evaluating its own line
        auto run_group = [&](int g0, int g1) {
            const int gi = g0 + lane;
            float dl = 0.f, f = 0.f, inva = 0.f, nfa = 0.f, xl = -1.f, cK = 0.f, y = 1.f, y2 = 1.f;
            int type = kLaneNone;
            float clo = 1e9f, chi = -1e9f;
            if (gi < g1) {
                const int li = order[gi];
                const float4 A = poolA[li], B = poolB[li];
                dl = A.x; f = A.y; inva = A.z; xl = A.w; cK = B.x; y2 = B.y; type = __float_as_int(B.z);
                nfa = __fmul_rn(-f, inva);                                 // as gather_kernel rounds it
                y = sqrtf(y2);
                const float hw = sqrtf(xl) / inva + 1.0f;                  // |t| < hw covers every X < xl
                const float pos = dl + f;
                const float lo = fmaxf(ceilf(pos - hw), 0.f), hi = fminf(floorf(pos + hw), whi);
                if (hi >= lo) { clo = lo; chi = hi; }
            }
            float bmin = clo, bmax = chi;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                bmin = fminf(bmin, __shfl_xor_sync(0xffffffffu, bmin, o));
                bmax = fmaxf(bmax, __shfl_xor_sync(0xffffffffu, bmax, o));
            }
            if (bmax < bmin) return;
            TrapLine TL = trap_line(type == kLaneTrap ? y : 1.0f);   // what the trapezoid rule needs of the line alone
            asm volatile("" : "+f"(TL.ie), "+f"(TL.amp0));           // (kept in registers: not recomputed per bin)
            // groups are sorted by evaluator: when every live lane of the group runs the trapezoid rule (the common case) the
            // bin loop is compiled without the dispatch
            const bool all_trap = !kBinned && __all_sync(0xffffffffu, type == kLaneTrap || type == kLaneNone);
            const int b_end = (int)bmax;
            const int col = lane & (kStage - 1), half = lane >> 4;
            auto bins = [&](auto trap_only) {
                constexpr bool kTrapOnly = decltype(trap_only)::value;
#pragma unroll 1
                for (int b0 = (int)bmin; b0 <= b_end; b0 += kStage) {
                    const int ns = min(kStage, b_end - b0 + 1);              // steps of this block (warp-uniform)
                    float d = (float)b0 - dl;                                // exact (small integers)
#pragma unroll 2
                    for (int s = 0; s < ns; ++s, d += 1.0f) {
                        const float un = __fmaf_rn(d, inva, nfa);            // the row pass's u and X, bit for bit
                        const float X = __fmul_rn(un, un);
                        float val = 0.f;
                        if (X < xl) {
                            if (kTrapOnly) val = cK * trap_K<true>(fabsf(un), TL, wsh);
                            else val = kBinned ? cK * binned_K(d, f, y2, inva) : lane_value(type, cK, fabsf(un), X, y, y2, TL, wsh);
                        }
                        stage[warp][s][lane] = val;
                    }
                    __syncwarp();
                    float sum = 0.f;
                    if (col < ns) {
#pragma unroll
                        for (int j = 0; j < 16; ++j) sum += stage[warp][col][half * 16 + j];
                    }
                    sum += __shfl_xor_sync(0xffffffffu, sum, 16);
                    if (half == 0 && col < ns) sacc[warp][b0 + col] += sum;
                    __syncwarp();
                }
            };
            if (all_trap) bins(std::true_type());
            else bins(std::false_type());
            since_flush += 32;     // the bin tile holds at most 32 lines' terms per bin per group
            if (since_flush >= kFlush) flush();
        };
        // sort the pool by evaluator (lines that are neighbours in centre-bin order have nearly the same centre and Doppler
        // width, so the 32 lines of a group also share ring position and width) and work it off
        auto run_pool = [&](int n, bool final) {
            int cls[kPPT], rk[kPPT];
            if (threadIdx.x < kYClasses) hist[threadIdx.x] = 0;
            if (threadIdx.x == 0) s_next = 0;
            __syncthreads();
#pragma unroll
            for (int k = 0; k < kPPT; ++k) {
                const int i = threadIdx.x + k * kThreads;
                cls[k] = -1;
                if (i < n) {
                    const float4 B = poolB[i];
                    cls[k] = kBinned ? 0 : __float_as_int(B.z);            // the evaluator (kLane*)
                    rk[k] = atomicAdd(&hist[cls[k]], 1);
                }
            }
            __syncthreads();
            const int cnt = hist[lane];
            int inc = cnt;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int up = __shfl_up_sync(0xffffffffu, inc, o);
                if (lane >= o) inc += up;
            }
#pragma unroll
            for (int k = 0; k < kPPT; ++k) {
                const int off = __shfl_sync(0xffffffffu, inc - cnt, cls[k] >= 0 ? cls[k] : 0);
                if (cls[k] >= 0) order[off + rk[k]] = (unsigned short)(threadIdx.x + k * kThreads);
            }
            __syncthreads();
            // only FULL groups are worked off before the unit's last pool: the remainder (< 32 lines, the tail of the sorted
            // order) goes back to the front of the pool and waits for company
            const int n_grp = final ? (n + 31) >> 5 : n >> 5;
            for (;;) {
                int grp = 0;
                if (lane == 0) grp = atomicAdd(&s_next, 1);
                grp = __shfl_sync(0xffffffffu, grp, 0);
                if (grp >= n_grp) break;
                run_group(32 * grp, min(32 * grp + 32, n));
            }
            const int rest = final ? 0 : n - 32 * n_grp;
            float4 keepA = make_float4(0.f, 0.f, 0.f, 0.f), keepB = keepA;
            if ((int)threadIdx.x < rest) { const int li = order[32 * n_grp + threadIdx.x]; keepA = poolA[li]; keepB = poolB[li]; }
            __syncthreads();
            if ((int)threadIdx.x < rest) { poolA[threadIdx.x] = keepA; poolB[threadIdx.x] = keepB; }
            if (threadIdx.x == 0) s_pool_n = rest;
        };

        if (threadIdx.x == 0) s_pool_n = 0;
        fetch(0);
        for (int v0 = 0; v0 < nt; v0 += kSubC) {
            __syncthreads();                        // s_pool_n settled; the pool is free to append to
#pragma unroll
            for (int k = 0; k < kLPTC; ++k) {
                if (v0 + threadIdx.x + k * kThreads < nt) {
                    const CentreLine L = centre_setup<KB>(preA[k], preC[k], ct0, a.profile);
                    if (L.lane != kLaneNone) {
                        const int slot = atomicAdd(&s_pool_n, 1);
                        poolA[slot] = make_float4(-L.ndl, -L.nf, L.inva, L.xl);
                        poolB[slot] = make_float4(preK[k], kBinned ? L.flo : L.y2, __int_as_float(L.lane), 0.f);
                    }
                }
            }
            __syncthreads();
            if (v0 + kSubC < nt) fetch(v0 + kSubC);
            const int n = s_pool_n;
            const bool last = v0 + kSubC >= nt;
            if (n > kCap - kSubC || (last && n > 0)) { any_work = true; run_pool(n, last); }
        }
        flush();
        __syncthreads();               // every warp is done with the staging matrix: red may overwrite it
        if (any_work) flush_tile<KB, W>(red, acc64, ct0, a);     // (uniform: every warp saw the same pool sizes)
    }
}

}  // namespace hk
