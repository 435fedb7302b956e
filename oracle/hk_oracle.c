/*
 * hk_oracle.c -- plain fp64 CPU ORACLE for the line-by-line opacity path of
 * HELIOS-K 2.0 (arxiv 2101.02005; citations are PAPER.md lines).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, bench.py's
 * cpu_baseline / --impl reference legs and __graft_entry__.smoke() may call
 * it.  It shares no code, header, table or constant with the CUDA library in
 * paper_2101_02005_b200/csrc/ and neither includes the other.
 *
 * What it computes is the *definition* of the result, by brute force:
 *
 *   k(nu_i) = sum over lines l with i_lo(l) <= i <= i_hi(l) of
 *             S_l * Re w(x + i y) / (alpha_D,l * sqrt(pi))
 *   x = (nu_i - nu0_l)/alpha_D,l   (Eq. 11)
 *   y = Gamma_L,l/alpha_D,l        (Eq. 12)
 *   alpha_D = (nu0/c) sqrt(2 k_B T/m)                        (Eq. 13; Eq. 3)
 *   Gamma_L = A/(4 pi c) + gamma_ref (T_ref/T)^n (P/P_ref)   (Eq. 5)
 *   S = A g'/(8 pi c m nu0^2 Q) exp(-c2 E''/T) (1 - exp(-c2 nu0/T))   (Eq. 9)
 *   nu_i = numin + i*dnu, i = 0..N-1  (Eq. 14: constant resolution)
 *   cut measured from the line centre (L239, L262); no cut for atoms (L7).
 *
 * Readings where the paper is silent or garbled are DESIGN.md "Readings" R1-R18
 * (normalisation of voigt(x,y): unit area in nu, R1; CODATA constants, R2/R3;
 * T_ref = 296 K and P_ref = 1 atm, R5; inclusive integer extents, R7; grid
 * size rounding, R8; point sampling, R9; nu0 <= 0 or non-finite => skipped, R14;
 * expm1 for the stimulated-emission factor, R15).
 *
 * Re w(z) is evaluated by the trapezoid rule on the convolution integral
 *   K(x,y) = (y/pi) Int exp(-t^2)/((x-t)^2+y^2) dt
 * with the residue correction for the pole at t = z (Matta & Reichel 1971,
 * Hunter & Regan 1972), h = 1/2, nodes n = -14..14; truncation error
 * O(exp(-pi^2/h^2)) ~ 1e-17.  The paper evaluates region C with Algorithm 916
 * (L156), which is "up to machine precision" (L146): any machine-precision
 * w(z) is the definition.  Pinned in tests/test_oracle_faddeeva.py against
 * numerical quadrature, erfcx, the Gaussian/Lorentzian limits and the
 * asymptotic series.  y == 0 is the pure Gaussian exp(-x^2).
 * Known limit: when x sits on or next to a node and y -> 0 the node's term
 * and the pole term cancel like h/(pi y); the phase of the pole term is
 * formed from the distance to the nearest node, which keeps the relative
 * accuracy at ~1e-16 h/(pi y) (pinned on and around the nodes down to
 * y = 1e-10 in tests/test_oracle_faddeeva.py: P = 0 leaves natural widths
 * only, y ~ 1e-9).
 *
 * Pins (tests/test_oracle_*.py, all `-m "not gpu"`): w(z) as above; profile
 * area, limits and wing loss; S by a decimal hand calculation, scaling laws and
 * the integrated-opacity identity; extents by brute force over bins; the sum by
 * linearity, permutation invariance and a 3-line x 11-bin case written out.
 * The paper prints no value of k(nu): beyond those pins the whole-spectrum
 * result is "parity unpinned" by any external number.
 *
 * Build: gcc -O2 -fopenmp -ffp-contract=off -shared -fPIC (see oracle/build.py).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* CODATA 2018 exact values, cgs (R2, R3). c as printed at L129. */
static const double HKO_C    = 2.99792458e10;   /* cm/s */
static const double HKO_KB   = 1.380649e-16;    /* erg/K */
static const double HKO_H    = 6.62607015e-27;  /* erg s */
static const double HKO_NA   = 6.02214076e23;   /* 1/mol */
static const double HKO_TREF = 296.0;           /* K, config 1 of BASELINE.json */
static const double HKO_PI   = 3.14159265358979323846;

int hko_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ---- Re w(x+iy), y >= 0 ------------------------------------------------ */
/* trapezoid weights exp(-(n h)^2), n = -14..14, h = 1/2; filled once at load */
#define HKO_NNODE 14
static double hko_wt[2 * HKO_NNODE + 1];
__attribute__((constructor)) static void hko_init_weights(void)
{
    for (int n = -HKO_NNODE; n <= HKO_NNODE; ++n) {
        double t = n * 0.5;
        hko_wt[n + HKO_NNODE] = exp(-t * t);
    }
}

double hko_voigt_K(double x, double y)
{
    const double h = 0.5;
    if (y == 0.0) return exp(-x * x);               /* pure Doppler limit */
    double s = 0.0;
    for (int n = -HKO_NNODE; n <= HKO_NNODE; ++n) {
        double t = n * h;
        double d = x - t;
        s += hko_wt[n + HKO_NNODE] / (d * d + y * y);
    }
    double K = h * y / HKO_PI * s;
    double re2 = x * x - y * y;
    if (y < HKO_PI / h && re2 < 700.0) {
        /* + Re{ 2 exp(-z^2) / (1 - exp(-2 pi i z/h)) },  z = x + i y */
        double amp = 2.0 * exp(-re2);
        double phi = 2.0 * x * y;                   /* exp(-z^2) = e^{-re2} (cos phi - i sin phi) */
        double nr = amp * cos(phi), ni = -amp * sin(phi);
        double em1 = expm1(2.0 * HKO_PI * y / h);   /* e - 1, e = exp(2 pi y/h) */
        /* exp(-2 pi i z/h) = e (cos th - i sin th), th = 2 pi x/h.  It has period h in x, so th is formed from the
         * distance to the NEAREST node (an exact subtraction), not from x: next to a node and for y of the same size
         * as that distance the pole term and the node's term are both ~h/(pi y) and must cancel to full precision,
         * which the rounding of 2 pi x/h (1e-16 x 4 pi x absolute) would spoil */
        double xr = x - h * nearbyint(x / h);
        double th = 2.0 * HKO_PI * xr / h;
        double sh = sin(0.5 * th);
        /* 1 - e cos th written as 2 sin^2(th/2) - (e-1) cos th: no cancellation
         * when x is on a node (th = 2 pi n) and y is small */
        double dr = 2.0 * sh * sh - em1 * cos(th), di = (1.0 + em1) * sin(th);
        K += (nr * dr + ni * di) / (dr * dr + di * di);
    }
    return K;
}

void hko_voigt_K_array(int64_t n, const double *x, const double *y, double *out)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) out[i] = hko_voigt_K(x[i], y[i]);
}

/* ---- grid ----------------------------------------- */
int64_t hko_grid_size(double numin, double numax, double dnu)
{
    return (int64_t)floor((numax - numin) / dnu + 0.5);
}

/* ---- per-line parameters (Eq. 13, 5, 9) -------------------------------- */
static int line_valid(double nu0, double A, double g, double E, double gam, double nx)
{
    return isfinite(nu0) && isfinite(A) && isfinite(g) && isfinite(E) && isfinite(gam) &&
           isfinite(nx) && nu0 > 0.0 && A >= 0.0;
}

static void line_params(double nu0, double A, double g, double E, double gam, double nx,
                        double T, double P_atm, double mass_amu, double Q,
                        double *S, double *gammaL, double *alphaD)
{
    double m = mass_amu / HKO_NA;                                   /* grams, L83 */
    double c2 = HKO_H * HKO_C / HKO_KB;                             /* cm K */
    *alphaD = (nu0 / HKO_C) * sqrt(2.0 * HKO_KB * T / m);           /* Eq. 13 inverted */
    *gammaL = A / (4.0 * HKO_PI * HKO_C) + gam * pow(HKO_TREF / T, nx) * P_atm;   /* Eq. 5 */
    *S = A * g / (8.0 * HKO_PI * HKO_C * m * nu0 * nu0 * Q)
         * exp(-c2 * E / T) * (-expm1(-c2 * nu0 / T));             /* Eq. 9 */
}

void hko_line_params(int64_t n, const double *nu0, const double *A, const double *g,
                     const double *E, const double *gam, const double *nx,
                     double T, double P_atm, double mass_amu, double Q,
                     double *S, double *gammaL, double *alphaD, int32_t *valid)
{
#pragma omp parallel for schedule(static)
    for (int64_t l = 0; l < n; ++l) {
        int v = line_valid(nu0[l], A[l], g[l], E[l], gam[l], nx[l]);
        valid[l] = v;
        if (v) line_params(nu0[l], A[l], g[l], E[l], gam[l], nx[l], T, P_atm, mass_amu, Q,
                           &S[l], &gammaL[l], &alphaD[l]);
        else { S[l] = 0.0; gammaL[l] = 0.0; alphaD[l] = 0.0; }
    }
}

/* ---- integer extents ------------------------------- */
/* cut > 0 and finite: fixed cutting length from the centre; otherwise uncut. */
static void line_extent(double nu0, double numin, double dnu, int64_t N, double cut,
                        int64_t *ilo, int64_t *ihi, int64_t *jc)
{
    const double big = 4.0e18;
    double c = floor((nu0 - numin) / dnu);
    if (c > big) c = big;
    if (c < -big) c = -big;
    *jc = (int64_t)c;
    if (cut > 0.0 && isfinite(cut)) {
        double lo = ceil((nu0 - cut - numin) / dnu);
        double hi = floor((nu0 + cut - numin) / dnu);
        if (lo < 0.0) lo = 0.0;
        if (hi > (double)(N - 1)) hi = (double)(N - 1);
        if (lo > big) lo = big;
        if (hi < -big) hi = -big;
        *ilo = (int64_t)lo;
        *ihi = (int64_t)hi;
    } else {
        *ilo = 0;
        *ihi = N - 1;
    }
}

/* invalid lines get the empty extent [0,-1] and jc = 0 */
void hko_extents(int64_t n, const double *nu0, const int32_t *valid, double numin, double dnu,
                 int64_t N, double cut, int64_t *ilo, int64_t *ihi, int64_t *jc)
{
#pragma omp parallel for schedule(static)
    for (int64_t l = 0; l < n; ++l) {
        if (valid && !valid[l]) { ilo[l] = 0; ihi[l] = -1; jc[l] = 0; continue; }
        line_extent(nu0[l], numin, dnu, N, cut, &ilo[l], &ihi[l], &jc[l]);
    }
}

/* ---- one line's profile value at wavenumber nu (unit area in nu, R1) ---- */
double hko_profile(double nu, double nu0, double gammaL, double alphaD)
{
    double x = (nu - nu0) / alphaD;
    double y = gammaL / alphaD;
    return hko_voigt_K(x, y) / (alphaD * sqrt(HKO_PI));
}

/* ---- k at a list of bins: brute force over lines [l0, l1) ---------------
 * Membership is decided by the integer extent only.  l0/l1 let a caller that
 * KNOWS no other line can reach these bins (centres sorted, fixed cut) skip
 * them; passing 0, n is the definition.  Neumaier-compensated sum per bin.
 * evals_out (optional) receives the number of (line, bin) evaluations. */
/* The selectable line profiles of section 2.1 (L47), each of unit area in nu, as a shape K with V = K/(alpha_D sqrt(pi)):
 *   0 Voigt    K = Re w(x + i y)
 *   1 Lorentz  V = Gamma_L/(pi ((nu - nu0)^2 + Gamma_L^2))          => K = y/(sqrt(pi) (x^2 + y^2))
 *   2 Doppler  V = exp(-x^2)/(alpha_D sqrt(pi))                      => K = exp(-x^2)
 *   3 binned Gaussian: the Doppler profile averaged over each bin (see below) */
static double shape_K(int profile, double x, double y, double hx)
{
    if (profile == 1) return y / (sqrt(HKO_PI) * (x * x + y * y));
    if (profile == 2) return exp(-x * x);
    if (profile == 3) {
        /* "binned Gaussian integrated cross section" of ExoCross (L47; PAPER.md prints no formula: DESIGN.md R26):
         * the Doppler profile averaged over the bin [nu_i - dnu/2, nu_i + dnu/2],
         *   V_i = (1/(2 dnu)) [erf(x + hx) - erf(x - hx)],  hx = dnu/(2 alpha_D)  =>  K = V alpha_D sqrt(pi).
         * erfc in the tails, where the two erf are both within rounding of 1. */
        double u = fabs(x), lo = u - hx, hi = u + hx;
        double d = lo >= 0.0 ? erfc(lo) - erfc(hi) : erf(hi) - erf(lo);
        return sqrt(HKO_PI) / (4.0 * hx) * d;
    }
    return hko_voigt_K(x, y);
}

/* plinth != 0 (and a finite cut): every term is S (V(nu_i - nu0) - V(cut)), the line with its "plinth" -- its own
 * value at the cutting length position -- removed from every bin of its extent (section 2.1.1; DESIGN.md
 * R21: the plinth is the profile AT nu0 +- cut, not at the last grid point inside the extent). */
void hko_opacity_bins_ex(int64_t n, const double *nu0, const double *A, const double *g,
                         const double *E, const double *gam, const double *nx,
                         double T, double P_atm, double mass_amu, double Q,
                         double numin, double dnu, int64_t N, double cut, int plinth, int profile,
                         int cut_mode, int64_t nb, const int64_t *bins, int64_t l0, int64_t l1,
                         double *k_out, int64_t *evals_out);

void hko_opacity_bins(int64_t n, const double *nu0, const double *A, const double *g,
                      const double *E, const double *gam, const double *nx,
                      double T, double P_atm, double mass_amu, double Q,
                      double numin, double dnu, int64_t N, double cut,
                      int64_t nb, const int64_t *bins, int64_t l0, int64_t l1,
                      double *k_out, int64_t *evals_out)
{
    hko_opacity_bins_ex(n, nu0, A, g, E, gam, nx, T, P_atm, mass_amu, Q, numin, dnu, N, cut, 0, 0, 0, nb, bins, l0, l1,
                        k_out, evals_out);
}

void hko_opacity_bins_ex(int64_t n, const double *nu0, const double *A, const double *g,
                         const double *E, const double *gam, const double *nx,
                         double T, double P_atm, double mass_amu, double Q,
                         double numin, double dnu, int64_t N, double cut, int plinth, int profile,
                         int cut_mode, int64_t nb, const int64_t *bins, int64_t l0, int64_t l1,
                         double *k_out, int64_t *evals_out)
{
    int64_t nl = l1 - l0;
    if (nl < 0) nl = 0;
    double *S = (double *)malloc(sizeof(double) * (size_t)(nl + 1));
    double *gL = (double *)malloc(sizeof(double) * (size_t)(nl + 1));
    double *aD = (double *)malloc(sizeof(double) * (size_t)(nl + 1));
    int64_t *ilo = (int64_t *)malloc(sizeof(int64_t) * (size_t)(nl + 1));
    int64_t *ihi = (int64_t *)malloc(sizeof(int64_t) * (size_t)(nl + 1));
    double *pl = (double *)malloc(sizeof(double) * (size_t)(nl + 1));   /* V(cut) per line, 0 without plinth removal */
    const int use_plinth = plinth && cut > 0.0 && isfinite(cut);
    (void)n;
#pragma omp parallel for schedule(static)
    for (int64_t q = 0; q < nl; ++q) {
        int64_t l = l0 + q, jc;
        if (line_valid(nu0[l], A[l], g[l], E[l], gam[l], nx[l])) {
            line_params(nu0[l], A[l], g[l], E[l], gam[l], nx[l], T, P_atm, mass_amu, Q,
                        &S[q], &gL[q], &aD[q]);
            /* cutting length of this line (L239: "a fixed cutting length, a fraction of the Doppler half-width, or a
             * fraction of the Lorentzian half-width"; R25): cut_mode 0: cut in cm^-1; 1: cut x Gamma_L;
             * 2: cut x Gamma_D, Gamma_D = alpha_D sqrt(ln 2) (L193-206) */
            double cl = cut;
            if (cut > 0.0 && isfinite(cut)) {
                if (cut_mode == 1) cl = cut * gL[q];
                else if (cut_mode == 2) cl = cut * aD[q] * sqrt(log(2.0));
            }
            if ((cut_mode == 1 || cut_mode == 2) && cut > 0.0 && isfinite(cut) && !(cl > 0.0)) {
                ilo[q] = 0; ihi[q] = -1;                       /* zero width: the line has no extent */
                pl[q] = 0.0;
            } else {
                line_extent(nu0[l], numin, dnu, N, cl, &ilo[q], &ihi[q], &jc);
                pl[q] = use_plinth ? shape_K(profile, cl / aD[q], gL[q] / aD[q], dnu / (2.0 * aD[q])) : 0.0;
            }
        } else { S[q] = 0.0; gL[q] = 0.0; aD[q] = 1.0; ilo[q] = 0; ihi[q] = -1; pl[q] = 0.0; }
    }
    int64_t evals = 0;
    const double sqrtpi = sqrt(HKO_PI);
#pragma omp parallel for schedule(dynamic, 1) reduction(+ : evals)
    for (int64_t b = 0; b < nb; ++b) {
        int64_t i = bins[b];
        double nu = numin + (double)i * dnu;
        double sum = 0.0, comp = 0.0;
        for (int64_t q = 0; q < nl; ++q) {
            if (i < ilo[q] || i > ihi[q]) continue;
            double x = (nu - nu0[l0 + q]) / aD[q];
            double y = gL[q] / aD[q];
            double term = S[q] * (shape_K(profile, x, y, dnu / (2.0 * aD[q])) - pl[q]) / (aD[q] * sqrtpi);
            double t = sum + term;                 /* Neumaier */
            if (fabs(sum) >= fabs(term)) comp += (sum - t) + term;
            else comp += (term - t) + sum;
            sum = t;
            ++evals;
        }
        k_out[b] = sum + comp;
    }
    if (evals_out) *evals_out = evals;
    free(S); free(gL); free(aD); free(ilo); free(ihi); free(pl);
}

/* ---- HITRAN-style inputs --------------------------------------------
 * Per line: nu0, A, g', E'', gamma_air, gamma_self, n, delta (Table 3-4) and an isotopologue index into a
 * table of (mass, Q(T), abundance) (species parameter file, L371-373, Table 2).
 *   Gamma_L = A/(4 pi c) + (T/T_ref)^-n [gamma_air (P - P_self)/P_ref + gamma_self P_self/P_ref]        (Eq. 4)
 *   centre  = nu0 + delta P      (pressure shift, L238, Table 4 "pressure-dependent line shift", cm^-1/atm; R23:
 *                                 the profile and the extent are centred there, S and alpha_D use the tabulated nu0)
 *   alpha_D = (nu0/c) sqrt(2 k_B T/m_iso),  S = abundance_iso x Eq. 9 with m_iso and Q_iso               (R24)
 * A line with an isotopologue index outside the table, or a non-finite field, contributes nothing (R14). */
static int line_valid_hitran(double nu0, double A, double g, double E, double ga, double gs, double nx, double dl,
                             int32_t iso, int32_t n_iso)
{
    return isfinite(nu0) && isfinite(A) && isfinite(g) && isfinite(E) && isfinite(ga) && isfinite(gs) &&
           isfinite(nx) && isfinite(dl) && nu0 > 0.0 && A >= 0.0 && iso >= 0 && iso < n_iso;
}

void hko_line_params_hitran(int64_t n, const double *nu0, const double *A, const double *g, const double *E,
                            const double *ga, const double *gs, const double *nx, const double *dl, const int32_t *iso,
                            double T, double P_atm, double P_self, int32_t n_iso, const double *mass_amu,
                            const double *Q, const double *abund,
                            double *S, double *gammaL, double *alphaD, double *centre, int32_t *valid)
{
    const double c2 = HKO_H * HKO_C / HKO_KB;
#pragma omp parallel for schedule(static)
    for (int64_t l = 0; l < n; ++l) {
        int v = line_valid_hitran(nu0[l], A[l], g[l], E[l], ga[l], gs[l], nx[l], dl[l], iso[l], n_iso);
        valid[l] = v;
        S[l] = 0.0; gammaL[l] = 0.0; alphaD[l] = 0.0; centre[l] = 0.0;
        if (!v) continue;
        const double m = mass_amu[iso[l]] / HKO_NA;
        alphaD[l] = (nu0[l] / HKO_C) * sqrt(2.0 * HKO_KB * T / m);
        gammaL[l] = A[l] / (4.0 * HKO_PI * HKO_C)
                    + pow(T / HKO_TREF, -nx[l]) * (ga[l] * (P_atm - P_self) + gs[l] * P_self);     /* P_ref = 1 atm */
        S[l] = abund[iso[l]] * A[l] * g[l] / (8.0 * HKO_PI * HKO_C * m * nu0[l] * nu0[l] * Q[iso[l]])
               * exp(-c2 * E[l] / T) * (-expm1(-c2 * nu0[l] / T));
        centre[l] = nu0[l] + dl[l] * P_atm;
    }
}

/* k at the listed bins from already computed per-line parameters: the same brute-force sum as hko_opacity_bins
 * (membership by the integer extent of the shifted centre, Neumaier-compensated). */
void hko_opacity_bins_params(int64_t n, const double *centre, const double *S, const double *gammaL,
                             const double *alphaD, const int32_t *valid, double numin, double dnu, int64_t N, double cut,
                             int64_t nb, const int64_t *bins, double *k_out, int64_t *evals_out)
{
    int64_t *ilo = (int64_t *)malloc(sizeof(int64_t) * (size_t)(n + 1));
    int64_t *ihi = (int64_t *)malloc(sizeof(int64_t) * (size_t)(n + 1));
#pragma omp parallel for schedule(static)
    for (int64_t l = 0; l < n; ++l) {
        int64_t jc;
        if (valid[l]) line_extent(centre[l], numin, dnu, N, cut, &ilo[l], &ihi[l], &jc);
        else { ilo[l] = 0; ihi[l] = -1; }
    }
    int64_t evals = 0;
    const double sqrtpi = sqrt(HKO_PI);
#pragma omp parallel for schedule(dynamic, 1) reduction(+ : evals)
    for (int64_t b = 0; b < nb; ++b) {
        int64_t i = bins[b];
        double nu = numin + (double)i * dnu;
        double sum = 0.0, comp = 0.0;
        for (int64_t l = 0; l < n; ++l) {
            if (i < ilo[l] || i > ihi[l]) continue;
            double term = S[l] * hko_voigt_K((nu - centre[l]) / alphaD[l], gammaL[l] / alphaD[l]) / (alphaD[l] * sqrtpi);
            double t = sum + term;
            if (fabs(sum) >= fabs(term)) comp += (sum - t) + term;
            else comp += (term - t) + sum;
            sum = t;
            ++evals;
        }
        k_out[b] = sum + comp;
    }
    if (evals_out) *evals_out = evals;
    free(ilo); free(ihi);
}
