// hk_device.cuh -- constants, record layouts and the fp32 Voigt evaluator shared by the
// CUDA kernels of the line-by-line opacity path (HELIOS-K 2.0, arxiv 2101.02005).
// Nothing here is shared with oracle/ (separate constants, separate formulas).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/hk.h"

namespace hk {

// ---- physical constants, cgs (CODATA 2018; c as printed in PAPER.md L129; R2/R3)
constexpr double kC = 2.99792458e10;     // cm/s
constexpr double kKB = 1.380649e-16;     // erg/K
constexpr double kH = 6.62607015e-27;    // erg s
constexpr double kNA = 6.02214076e23;    // 1/mol
constexpr double kTref = 296.0;          // K (Eq. 5; BASELINE.json config 1)
constexpr double kPi = 3.141592653589793238462643383279502884;

// ---- geometry of the accumulation kernels (KB = bins per lane is a template parameter: 2, 4 or 8)
constexpr int kWarps = 8;                // warps per CTA
constexpr int kThreads = 32 * kWarps;
constexpr int kSub = 512;                // line records staged in shared memory at a time
constexpr int kFlush = 128;              // fp32 partial sums hold at most this many lines
// interior (mask-free) kernels only see |t| >= 2*KB bins: with the centre position held as ONE fp32
// relative to the tile (|tl| <= 32 KB + |t|) the rounding of t stays below 2^-24 (1 + 16) |t| = 1.0e-6 |t|
constexpr int kMinDistPerKB = 2;

constexpr int32_t kKeySentinelBias = 1;  // sentinel key = kmax + 1

// ---- unsorted per-line record written by the preprocess kernel (32 B)
struct __align__(16) RecU {
    int32_t jc;      // centre bin floor((nu0-numin)/dnu)
    float f;         // sub-bin offset from the NEAREST grid point, [-1/2, 1/2]; sign bit set (-0 too): the point is jc + 1
    float G2;        // (Gamma_L/dnu)^2
    float a2;        // (alpha_D/dnu)^2
    int32_t ilo;     // inclusive integer extent
    int32_t ihi;
    double cK;       // S/(alpha_D sqrt(pi)) in cm^2/g per unit K (unscaled)
};

// sorted records consumed by the accumulation kernels: two float4 streams
//   A = { jp (int bits), f, G2, c }        centre = jp + f, jp the NEAREST grid point, f in [-1/2, 1/2];
//                                          c  = scale * S * Gamma_L/(pi dnu^2)   (Lorentz amplitude, bin units)
//   B = { a2, ilo (int bits), ihi (int bits), cK }   cK = scale * S/(alpha_D sqrt(pi))

//   N = { jc (int bits), (f13 << 19) | a2_19, G2, c }   compact record of the node kernel: f13 = sub-bin offset in
//       1/8192 bins, a2_19 = top 19 bits below the sign of the fp32 pattern of a2 (8 exponent + 11 mantissa bits)

// per level-0 tile: the candidate range [A0,A1) of sorted line indices and its split (hk_accumulate.cuh):
//   [A0,EL) left edge, no core | [EL,FL0) left edge, generic | [FL0,NL) node-handled | [NL,FL1) far | [FL1,ML1) mid |
//   [ML1,CL) centre, generic | [CL,CR) centre, tile inside the extent | [CR,MR0) centre, generic |
//   [MR0,FR0) mid | [FR0,NR) far | [NR,FR1) node-handled | [FR1,ER) right edge, generic | [ER,A1) right edge, no core
// [LL,LR) inside [CL,CR): the lines that can have innermost bins (lane-pass work, hk_centre.cuh) in this tile
struct __align__(8) TileRange {
    int32_t A0, EL, FL0, NL, FL1, ML1, CL, CR, MR0, FR0, NR, FR1, ER, A1, LL, LR;
};

// per (level, tile) entry of the node hierarchy: four index ranges of sorted lines evaluated at the tile's nodes
struct __align__(8) NodeRange {
    int32_t a0, a1, b0, b1, c0, c1, d0, d1;
    int32_t fL, fR;      // lines with index < fL (left ranges) or >= fR (right ranges) have |z|^2 >= Z1 on the whole tile:
                         // one asymptotic term is enough (the lists are sorted by centre, so far lines are a prefix / suffix)
    int32_t gL, gR;      // lines with gL <= index < gR may have |z|^2 < Z2 on the tile (the core at nodes): 4-point form
};

// ---- Chebyshev nodes of the separated-tile evaluation ----------------
constexpr int kP = HK_NODES;             // nodes per tile: degree-(kP-1) interpolant
constexpr int kMaxLevels = 24;
// xi_k = cos((2k+1) pi/(2 kP)); barycentric weights (-1)^k sin((2k+1) pi/(2 kP))
#if HK_NODES == 8
__device__ constexpr double kChebX[kP] = {0.98078528040323044913,  0.83146961230254523708,  0.55557023301960222474,
                                          0.19509032201612826785,  -0.19509032201612826785, -0.55557023301960222474,
                                          -0.83146961230254523708, -0.98078528040323044913};
__device__ constexpr double kChebW[kP] = {0.19509032201612826785,  -0.55557023301960222474, 0.83146961230254523708,
                                          -0.98078528040323044913, 0.98078528040323044913,  -0.83146961230254523708,
                                          0.55557023301960222474,  -0.19509032201612826785};
#elif HK_NODES == 10
__device__ constexpr double kChebX[kP] = {0.98768834059513772619,  0.89100652418836786236,  0.7071067811865475244,
                                          0.45399049973954679156,  0.15643446504023086901,  -0.15643446504023086901,
                                          -0.45399049973954679156, -0.7071067811865475244,  -0.89100652418836786236,
                                          -0.98768834059513772619};
__device__ constexpr double kChebW[kP] = {0.15643446504023086901,  -0.45399049973954679156, 0.7071067811865475244,
                                          -0.89100652418836786236, 0.98768834059513772619,  -0.98768834059513772619,
                                          0.89100652418836786236,  -0.7071067811865475244,  0.45399049973954679156,
                                          -0.15643446504023086901};
#elif HK_NODES == 12
__device__ constexpr double kChebX[kP] = {0.99144486137381041114,  0.92387953251128675613,  0.79335334029123516458,
                                          0.60876142900872063942,  0.38268343236508977173,  0.13052619222005159155,
                                          -0.13052619222005159155, -0.38268343236508977173, -0.60876142900872063942,
                                          -0.79335334029123516458, -0.92387953251128675613, -0.99144486137381041114};
__device__ constexpr double kChebW[kP] = {0.13052619222005159155,  -0.38268343236508977173, 0.60876142900872063942,
                                          -0.79335334029123516458, 0.92387953251128675613,  -0.99144486137381041114,
                                          0.99144486137381041114,  -0.92387953251128675613, 0.79335334029123516458,
                                          -0.60876142900872063942, 0.38268343236508977173,  -0.13052619222005159155};
#else
#error "HK_NODES must be 8, 10 or 12"
#endif

struct Levels {
    int32_t n_levels;                    // node levels 0..n_levels-1, tile width W0 << l
    int32_t w0;                          // level-0 tile width (32 kb)
    int32_t n_entries;                   // sum over levels of tiles
    int32_t off[kMaxLevels + 1];         // first entry of each level
};

// ---- small helpers
__device__ __forceinline__ float rcp_approx(float x)
{
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

// ---- fp32 evaluator, by region of |z|^2 = x^2 + y^2 ----------------
// All three work in "bin units": t = (nu_i - nu0)/dnu, G = Gamma_L/dnu, a = alpha_D/dnu,
// q = t^2 + G^2 = a^2 |z|^2.
//
// far  (|z|^2 >= HK_Z1): first term of the asymptotic series of w(z) = i/(sqrt(pi) z) (1 + 1/(2z^2) + ...)
//        S V = c / q                      -- the Lorentzian, what the paper's region A evaluates
//        with a first-order Gauss-Hermite rule (Table 1).
// mid  (HK_Z2 <= |z|^2 < HK_Z1): two terms,
//        S V = c r (1 + r (1.5 a^2 - 2 a^2 G^2 r)),  r = 1/q
//        since Re{ i/z (1 + 1/(2 z^2)) } = y/|z|^2 (1 + (3x^2 - y^2)/(2|z|^4)).
// core (|z|^2 < HK_Z2): trapezoid rule on the convolution integral with the pole term,
//        nodes shifted per evaluation so that x is never within h/4 of a node.
__device__ __forceinline__ float term_far(float c, float q) { return c * rcp_approx(q); }

__device__ __forceinline__ float shape_mid(float r, float A1, float A2)
{
    // r (1 + r (A1 - A2 r))
    float u = fmaf(-A2, r, A1);
    float v = fmaf(u, r, 1.0f);
    return r * v;
}

// core, outer rings (HK_Z3 <= |z|^2 < HK_Z2): n-point Gauss-Hermite quadrature of the convolution integral,
//        K = (y/pi) sum_k w_k / ((x - t_k)^2 + y^2)  (what the paper's regions A/B do with n = 1 and 3, Table 1
//        L148-159), with the symmetric node pairs +-t_k combined in real arithmetic:
//        1/((x-t)^2+y^2) + 1/((x+t)^2+y^2) = 2 A / (A^2 - 4 t^2 x^2),  A = x^2 + y^2 + t^2,
//        and all pairs brought over one denominator (one reciprocal per evaluation).
//        Measured against the oracle: n = 4 <= 1.0e-6 for |z| >= 8, n = 6 <= 7.7e-6 for |z| >= 5.5
//        (the floor is the exp(-x^2) part the quadrature cannot see; the trapezoid threshold rises to
//        |z|^2 < 50 for lines with y < 1e-3).
__device__ __forceinline__ float gh4_K(float x2, float s, float y)
{
    // nodes +-0.5246476232752903, +-1.650680123885785; weights 0.8049140900055128, 0.08131283544724518
    constexpr float T1 = 0.27525512860841095f, T2 = 2.7247448713915890f;      // t_k^2
    constexpr float W1 = 0.5124242247547685f, W2 = 0.05176535879298783f;       // 2 w_k / pi
    const float A1 = s + T1, A2 = s + T2;
    const float D1 = fmaf(A1, A1, (-4.0f * T1) * x2), D2 = fmaf(A2, A2, (-4.0f * T2) * x2);
    const float num = fmaf(W2 * A2, D1, (W1 * A1) * D2);
    return y * num * rcp_approx(D1 * D2);
}

__device__ __forceinline__ float gh6_K(float x2, float s, float y)
{
    // nodes +-0.4360774119276165, +-1.335849074013697, +-2.350604973674492;
    // weights 0.7246295952243925, 0.1570673203228566, 0.004530009905508846
    constexpr float T1 = 0.19016350919348813f, T2 = 1.7844927485432516f, T3 = 5.5253437422632603f;
    constexpr float W1 = 0.4613135279625653f, W2 = 0.09999216171032288f, W3 = 0.0028838938748679236f;   // 2 w_k / pi
    const float A1 = s + T1, A2 = s + T2, A3 = s + T3;
    const float D1 = fmaf(A1, A1, (-4.0f * T1) * x2), D2 = fmaf(A2, A2, (-4.0f * T2) * x2),
                D3 = fmaf(A3, A3, (-4.0f * T3) * x2);
    const float D12 = D1 * D2;
    float num = (W1 * A1) * (D2 * D3);
    num = fmaf(W2 * A2, D1 * D3, num);
    num = fmaf(W3 * A3, D12, num);
    return y * num * rcp_approx(D12 * D3);
}

// 10-point rule for the innermost region when the pole is far enough from the real axis: for y >= 1.8 the quadrature
// converges on all of |z|^2 < HK_Z3 (in fp64 against w(z): <= 8.2e-6, worst at y = 1.8, x = 0; 2.6e-6 from y = 2 on), at
// a quarter of the cost of the trapezoid evaluator with its pole term.
#define HK_Y10 1.8f
__device__ __forceinline__ float gh10_K(float x2, float s, float y)
{
    constexpr float T1 = 0.11758132021177813f, T2 = 1.074562012436904f, T3 = 3.0859374437175497f,
                    T4 = 6.41472973366203f, T5 = 11.807189489971735f;                       // t_k^2
    constexpr float W1 = 0.38888723083644433f, W2 = 0.15287698792389035f, W3 = 0.02156510928733804f,
                    W4 = 0.0008553914494585371f, W5 = 4.864050625087994e-06f;               // 2 w_k / pi
    const float A1 = s + T1, A2 = s + T2, A3 = s + T3, A4 = s + T4, A5 = s + T5;
    const float D1 = fmaf(A1, A1, (-4.0f * T1) * x2), D2 = fmaf(A2, A2, (-4.0f * T2) * x2),
                D3 = fmaf(A3, A3, (-4.0f * T3) * x2), D4 = fmaf(A4, A4, (-4.0f * T4) * x2),
                D5 = fmaf(A5, A5, (-4.0f * T5) * x2);
    float sum = fmaf(W2 * A2, D1, (W1 * A1) * D2) * rcp_approx(D1 * D2);
    sum = fmaf(fmaf(W4 * A4, D3, (W3 * A3) * D4), rcp_approx(D3 * D4), sum);
    sum = fmaf(W5 * A5, rcp_approx(D5), sum);
    return y * sum;
}

// The Gauss-Hermite rules converge faster the farther the pole lies from the real axis: the region each one is good
// for grows with y.  Measured in fp64 against the oracle's w(z) on a lattice (worst case always at the smallest |z|):
//   4 points: <= 3.0e-6 for |z|^2 >= 49 (any y), >= 36 (y >= 1.5), >= 30.25 (y >= 3); on ALL of the core for y >= 4.5 (5.7e-6)
//   6 points: <= 4.8e-7 for |z|^2 >= 30.25 (any y), <= 1.05e-6 for |z|^2 >= 21 (y >= 1); on ALL of the core for y >= 3 (3.6e-6)
//  10 points: on all of the core for y >= 1.8 (8.2e-6; y >= 2: 2.6e-6)
// so a line with y >= 4.5 -- the majority at high pressure -- has no inner rings at all.
#define HK_Y4 4.5f
#define HK_Y6 3.0f
// |z|^2 below which the 4-point rule is not used, as a function of y^2
__device__ __forceinline__ float z4_for(float y2)
{
    return y2 >= HK_Y4 * HK_Y4 ? 0.f : y2 >= HK_Y6 * HK_Y6 ? HK_Z3 : y2 >= 2.25f ? 36.0f : HK_Z4;
}
// |z|^2 below which the innermost evaluator is used, as a function of y^2
// (y = 0 exactly, the pure Gaussian of the Doppler profile: exp(-x^2) is ALL there is.  It is evaluated together with
//  its amplitude, gauss_term below, and followed down to x^2 = HK_ZG: with the launch scale putting the largest
//  amplitude at 2^100 that is the end of the fp32 range, 2^-126 -- DESIGN.md R22)
#define HK_ZG 157.0f
#define HK_ZN 49.0f          // the node hierarchy takes separated tiles with |z|^2 >= HK_ZN on all of them (4-point form valid for any y)
#define HK_Z3Y1 21.0f        // inner edge of the 6-point ring for y >= 1
__device__ __forceinline__ float z3_for(float y2)
{
    return y2 == 0.f ? HK_ZG : y2 >= HK_Y6 * HK_Y6 ? 0.f : y2 < 1e-6f ? 50.0f : y2 >= 1.0f ? HK_Z3Y1 : HK_Z3;
}

// cK exp(-x^2) for a pure Gaussian, amplitude and exponent combined BEFORE the exponential so that the product is
// followed to the end of the fp32 range even where exp(-x^2) alone would underflow (x^2 > 87).  The exponent is
// split so that its rounding error stays below 2^-22 up to x^2 = HK_ZG.
__device__ __forceinline__ float gauss_term(float cK, float x)
{
    constexpr float L2E_HI = 1.44269502162933349609375f;      // log2(e) = HI + LO
    constexpr float L2E_LO = 1.925963033500011e-08f;
    const float x2 = x * x;
    const float x2l = fmaf(x, x, -x2);                        // x^2 = x2 + x2l exactly
    const float p = x2 * L2E_HI;                              // x^2 log2(e) = p + e
    float e = fmaf(x2, L2E_HI, -p);
    e = fmaf(x2, L2E_LO, e);
    e = fmaf(x2l, L2E_HI, e);
    const float n = rintf(p);                                 // p - n is exact (p < 2^8)
    const float v = exp2f(n - p) * fmaf(-0.693147180559945f, e, 1.0f);
    // cK v 2^-n in two steps: 2^-n alone may lie below the fp32 range while the product does not
    const int k = min((int)n, 250), k1 = k >> 1;
    const float s1 = __int_as_float((127 - k1) << 23), s2 = __int_as_float((127 - (k - k1)) << 23);
    return ((cK * s1) * v) * s2;
}

// Re w(x + i y) for |z|^2 < HK_Z2, x >= 0, y > 0: ring by |z|^2
__device__ __forceinline__ float core_any_K(float x, float y, int* region);

// Re w(x + i y), x >= 0, 0 < y < 2 (< pi/h), intended for x^2 + y^2 < ~60.
// K = (h y/pi) sum_n exp(-t_n^2)/((x-t_n)^2 + y^2) + pole term, t_n = (n + s) h, h = 0.8, n = -5..5
// (Matta & Reichel 1971 / Hunter & Regan 1972: the family Algorithm 916, which the paper uses in region C
// (L156), belongs to).  Two node sets (s = 0, 1/2), chosen per evaluation so that x is never within h/4
// of a node.  The oracle uses h = 1/2, 29 nodes, fp64 and no node shift.
// Cost (the lane kernel is bound by instruction issue and by the special-function unit alike): the squared distances
// to the nodes are formed two at a time (packed fp32), THREE nodes share one reciprocal, and the pole term rides on
// the last reciprocal: 4 reciprocals per evaluation; everything that depends on y alone (TrapLine) is worked out once
// per line.  Pole term, with E = exp(-2 pi y/h) and theta = 2 pi (x/h - s):
//   Re{ 2 exp(-z^2) / (1 - exp(-2 pi i (z/h - s))) } = 2 exp(y^2 - 2 pi y/h) exp(-x^2) [cos(2xy)(E - cos theta) - sin(2xy) sin theta]
//                                                      / [(E - cos theta)^2 + sin^2 theta]
// (numerator and denominator divided by exp(4 pi y/h): nothing in it grows with y).
struct TrapLine {
    float y2, yk, ie, amp0, ty;        // y^2, y h/pi, exp(-2 pi y/h), 2 exp(y^2 - 2 pi y/h), 2 y
};
__device__ __forceinline__ TrapLine trap_line(float y)
{
    TrapLine L;
    L.y2 = y * y;
    L.yk = y * (0.8f / 3.14159265358979f);
    L.ie = __expf(-7.85398163f * y);                        // 2 pi/h = 7.854
    L.amp0 = 2.0f * __expf(fmaf(-7.85398163f, y, L.y2));
    L.ty = y + y;
    return L;
}
// weights exp(-((n+s)h)^2), n = -5..6 (the twelfth is there to make four triples; its weight is nil), s = 0 and s = 1/2
#define HK_TRAP_WA {1.12535175e-07f, 3.57128496e-05f, 3.15111160e-03f, 7.73047404e-02f, 5.27292424e-01f, 1.0f, \
                    5.27292424e-01f, 7.73047404e-02f, 3.15111160e-03f, 3.57128496e-05f, 1.12535175e-07f, 0.0f}
#define HK_TRAP_WB {2.35257520e-06f, 3.93669041e-04f, 1.83156389e-02f, 2.36927759e-01f, 8.52143789e-01f, 8.52143789e-01f, \
                    2.36927759e-01f, 1.83156389e-02f, 3.93669041e-04f, 2.35257520e-06f, 3.90893843e-09f, 0.0f}
// wtab: the 24 weights in shared memory (A then B; fill with trap_weights_to_shared), passed as their address in the
// shared window (trap_weights_address) -- or nullptr (selected from immediates)
__device__ __forceinline__ void trap_weights_to_shared(float* wtab, int tid)
{
    constexpr float wA[12] = HK_TRAP_WA, wB[12] = HK_TRAP_WB;
    if (tid < 12) wtab[tid] = wA[tid];
    else if (tid < 24) wtab[tid] = wB[tid - 12];
}
__device__ __forceinline__ const float* trap_weights_address(const float* wtab_shared)
{
    uint32_t a = (uint32_t)__cvta_generic_to_shared(wtab_shared);
    asm volatile("" : "+r"(a));                 // (kept in a register: not rebuilt per evaluation)
    return reinterpret_cast<const float*>((uintptr_t)a);
}
template <bool kSmemW>
__device__ __forceinline__ float trap_K(float x, const TrapLine& L, const float* __restrict__ wtab)
{
    constexpr float h = 0.8f, inv_h = 1.25f;
    const float u = x * inv_h;
    const float fr = u - floorf(u);
    const bool on = (fr >= 0.25f) && (fr < 0.75f);        // integer nodes are >= h/4 away
    const float s = on ? 0.0f : 0.5f;
    const float us = u - s;
    const float frs = us - floorf(us);                    // in [1/4, 3/4]
    const float xs = fmaf(-s, h, x);                      // x - s h
    // q_n = (xs - (n - 5) h)^2 + y^2, n = 0..11, two at a time
    float2 q[6];
    float2 d = make_float2(xs + 5.0f * h, xs + 4.0f * h);
    const float2 y2 = make_float2(L.y2, L.y2), step = make_float2(-2.0f * h, -2.0f * h);
    q[0] = __ffma2_rn(d, d, y2);
#pragma unroll
    for (int k = 1; k < 6; ++k) {
        d = __fadd2_rn(d, step);
        q[k] = __ffma2_rn(d, d, y2);                      // >= (h/4)^2
    }
    // w_a/q_a + w_b/q_b + w_c/q_c = (w_a q_b q_c + (w_b q_c + w_c q_b) q_a) / (q_a q_b q_c)
    float sum, num3, den3;
    {
        float4 w0, w1, w2;
        if (kSmemW) {
            // (wtab is a SHARED-window address here, formed once by the caller: the generic pointer made the compiler
            //  rebuild the window base, seven uniform instructions, at every evaluation)
            const uint32_t wa = (uint32_t)(uintptr_t)wtab + (on ? 0u : 48u);
            asm("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(w0.x), "=f"(w0.y), "=f"(w0.z), "=f"(w0.w) : "r"(wa));
            asm("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4+16];" : "=f"(w1.x), "=f"(w1.y), "=f"(w1.z), "=f"(w1.w) : "r"(wa));
            asm("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4+32];" : "=f"(w2.x), "=f"(w2.y), "=f"(w2.z), "=f"(w2.w) : "r"(wa));
        } else {
            constexpr float wA[12] = HK_TRAP_WA, wB[12] = HK_TRAP_WB;
            w0 = make_float4(on ? wA[0] : wB[0], on ? wA[1] : wB[1], on ? wA[2] : wB[2], on ? wA[3] : wB[3]);
            w1 = make_float4(on ? wA[4] : wB[4], on ? wA[5] : wB[5], on ? wA[6] : wB[6], on ? wA[7] : wB[7]);
            w2 = make_float4(on ? wA[8] : wB[8], on ? wA[9] : wB[9], on ? wA[10] : wB[10], 0.0f);
        }
#define HK_TRIPLE(qa, qb, qc, wa, wb, wc, num, den)                 \
        const float den##_bc = (qb) * (qc);                          \
        const float num = fmaf(fmaf((wb), (qc), (wc) * (qb)), (qa), (wa) * den##_bc); \
        const float den = (qa) * den##_bc;
        HK_TRIPLE(q[0].x, q[0].y, q[1].x, w0.x, w0.y, w0.z, n0, d0)
        HK_TRIPLE(q[1].y, q[2].x, q[2].y, w0.w, w1.x, w1.y, n1, d1)
        HK_TRIPLE(q[3].x, q[3].y, q[4].x, w1.z, w1.w, w2.x, n2, d2)
        HK_TRIPLE(q[4].y, q[5].x, q[5].y, w2.y, w2.z, w2.w, n3, d3)
#undef HK_TRIPLE
        sum = n0 * rcp_approx(d0);
        sum = fmaf(n1, rcp_approx(d1), sum);
        sum = fmaf(n2, rcp_approx(d2), sum);
        num3 = n3; den3 = d3;
    }
    // pole term over the last triple's denominator
    const float g = __expf(-x * x);
    const float phi = L.ty * x;                           // 2 x y, reduced to [-pi, pi] first
    const float kk = rintf(phi * 0.159154943f);
    float ph = fmaf(-kk, 6.28318548f, phi);
    ph = fmaf(-kk, -1.74845553e-07f, ph);                 // 2 pi = 6.28318548 - 1.74845553e-07
    float sp, cp;
    __sincosf(ph, &sp, &cp);
    // theta = 2 pi frac(x/h - s) in [pi/2, 3pi/2] (cos(theta) <= 0): theta - pi lies in [-pi/2, pi/2], where the
    // special-function unit's sin/cos are good to ~5e-7 absolute
    float st, ct;
    __sincosf(6.28318531f * (frs - 0.5f), &st, &ct);
    st = -st; ct = -ct;
    const float a = L.ie - ct;                            // >= exp(-2 pi y/h) > 0
    const float pn = (L.amp0 * g) * fmaf(cp, a, -sp * st);
    const float pd = fmaf(a, a, st * st);
    const float top = fmaf(L.yk * num3, pd, pn * den3);
    return fmaf(sum, L.yk, top * rcp_approx(den3 * pd));
}
__device__ __noinline__ float core_K(float x, float y) { return trap_K<false>(x, trap_line(y), nullptr); }

__device__ __forceinline__ float core_any_K(float x, float y, int* region)
{
    const float x2 = x * x, y2 = y * y, s = x2 + y2;
    if (y == 0.f) { if (region) *region = 4; return __expf(-x2); }     // pure Gaussian (with its amplitude: gauss_term)
    const float z3 = z3_for(y2);
    if (s >= fmaxf(z4_for(y2), z3)) { if (region) *region = 2; return gh4_K(x2, s, y); }
    if (s >= z3) { if (region) *region = 3; return gh6_K(x2, s, y); }
    if (y >= HK_Y10) { if (region) *region = 5; return gh10_K(x2, s, y); }
    if (region) *region = 4;
    return core_K(x, y);
}

// ---- binned Gaussian (HK_PROFILE_BINNED_GAUSSIAN): the Doppler profile averaged over the bin -------------------
// K = V alpha_D sqrt(pi) = (a sqrt(pi)/2) [erf(e_hi/a) - erf(e_lo/a)] in bin units (a = alpha_D/dnu), e_hi / e_lo the
// signed distances from the line centre to the bin's upper / lower edge; erfc in the tails; for a > 64 bins the
// second-order bin average exp(-x^2)(1 + h^2 (2 x^2 - 1)/3), h = 1/(2a), is exact to 1.4e-7 and avoids the
// cancellation of two nearly equal erfc.  Zero beyond |t| = 1/2 + 6 a.
// The edge distances come from the bin offset d = b - jp (an exact small integer) and the sub-bin offset of the centre
// as a hi/lo pair f + flo (R26): for a line much narrower than a bin whose centre lies within a few a of a
// bin edge, the share of the neighbouring bin depends on (1/2 - |f|)/a, which one fp32 f resolves to 2^-26/a only.
__device__ __forceinline__ float binned_K(float d, float f, float flo, float inv_a)
{
    if (inv_a < (1.0f / 64.0f)) {
        const float x = (d - f) * inv_a, h = 0.5f * inv_a;
        return __expf(-x * x) * fmaf(h * h * (1.0f / 3.0f), fmaf(2.0f * x, x, -1.0f), 1.0f);
    }
    // (d +- 1/2) - f is exact whenever the result is small (Sterbenz), which is when it matters
    const float lo = (((d - 0.5f) - f) - flo) * inv_a, hi = (((d + 0.5f) - f) - flo) * inv_a;
    const float dd = lo >= 0.f ? erfcf(lo) - erfcf(hi) : hi <= 0.f ? erfcf(-hi) - erfcf(-lo) : erff(hi) - erff(lo);
    return 0.886226925452758f * dd / inv_a;
}
__device__ __forceinline__ float binned_ql(float a2)
{
    const float h = fmaf(6.0f, sqrtf(a2), 0.5f);
    return h * h;
}
// S V of one (line, bin) pair where the row formulas do not apply, amplitude included: by profile.
// d = b - jp, t = d - f (the row pass's t), inv_a = dnu/alpha_D, y = Gamma_L/alpha_D, cK = scale S/(alpha_D sqrt(pi)).
__device__ __forceinline__ float core_term(int profile, float cK, float d, float f, float flo, float inv_a, float y)
{
    if (profile == HK_PROFILE_BINNED_GAUSSIAN) return cK * binned_K(d, f, flo, inv_a);
    const float x = fabsf(d - f) * inv_a;
    if (y == 0.f) return gauss_term(cK, x);
    return cK * core_any_K(x, y, nullptr);
}

}  // namespace hk
