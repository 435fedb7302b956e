/*
 * hk.h -- C ABI of the B200-native line-by-line opacity library
 * (hot path of HELIOS-K 2.0, arxiv 2101.02005; citations are PAPER.md lines).
 *
 * What the library computes:
 *
 *   k(nu_i) = sum over lines l with i_lo(l) <= i <= i_hi(l) of S_l * V_l(nu_i)
 *
 *   nu_i    = numin + i*dnu, i = 0..N-1, N = floor((numax-numin)/dnu + 0.5)   (Eq. 14)
 *   V_l     = Re w(x + i y) / (alpha_D sqrt(pi)),  x = (nu_i-nu0)/alpha_D, y = Gamma_L/alpha_D
 *                                                              (Eq. 1-2, Eq. 11-12)
 *   alpha_D = (nu0/c) sqrt(2 k_B T / m)                                      (Eq. 3, Eq. 13)
 *   Gamma_L = A/(4 pi c) + gamma_ref (T_ref/T)^n_exp (P/P_ref)               (Eq. 5)
 *   S_l     = A g'/(8 pi c m nu0^2 Q) exp(-c2 E''/T) (1 - exp(-c2 nu0/T))    (Eq. 9)
 *   cut     : fixed cutting length from the line centre (L239, L262), or none (atoms, L7)
 *
 * Units: cm^-1, K, atm, amu, s^-1; gamma_ref in cm^-1/atm at T_ref = 296 K,
 * P_ref = 1 atm; output cm^2 g^-1.  Constants: CODATA 2018 (c as printed at L129).
 *
 * All line arrays, the output and the workspace are DEVICE pointers owned by
 * the caller (PyTorch tensors in the Python binding).  The library owns only
 * the small host handle.  Inputs are never modified.  Every entry point returns
 * 0 on success or a negative hk_status; nothing throws, aborts or prints.
 * A context is not thread-safe.  There is no CPU fallback.
 */
#ifndef HK_H
#define HK_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct hk_ctx hk_ctx; /* opaque; one per grid */

typedef enum {
    HK_OK = 0,
    HK_EINVAL = -1, /* bad scalar, null pointer, n_lines < 0, N >= 2^31 - 2^12 */
    HK_ESTATE = -2, /* compute before conditions / workspace; get_* before a compute */
    HK_ENOSPC = -3, /* workspace smaller than hk_workspace_bytes() */
    HK_ECUDA = -4,  /* a CUDA call failed; raw code from hk_last_cuda_error() */
    HK_ENOMEM = -5  /* host allocation of the handle failed */
} hk_status;

/* Six SoA fp64 DEVICE arrays of n_lines elements each, read-only.
 * g_up holds integer values stored as fp64 (R18). */
typedef struct {
    const double* nu0;       /* line centre, cm^-1 */
    const double* A;         /* Einstein A, s^-1 */
    const double* g_up;      /* upper-state degeneracy g' */
    const double* E_low;     /* lower-state energy E'', cm^-1 */
    const double* gamma_ref; /* pressure-broadening coefficient at T_ref, cm^-1/atm */
    const double* n_exp;     /* temperature exponent n */
} hk_lines;

/* Exact integer work counts of the last hk_compute plus bookkeeping. */
typedef struct {
    int64_t n_lines;       /* as passed */
    int64_t n_skipped;     /* nu0 <= 0, A < 0 or a non-finite field: contribute nothing (R14) */
    int64_t n_off_grid;    /* valid lines whose extent misses the grid (or > 2^30 bins away) */
    int64_t n_evals;       /* sum over lines of (i_hi - i_lo + 1): Voigt evaluations */
    int64_t n_evals_far;   /* of those, |z|^2 >= HK_Z1 (1-term asymptotic = Lorentzian) */
    int64_t n_evals_mid;   /* HK_Z2 <= |z|^2 < HK_Z1 (2-term asymptotic) */
    int64_t n_evals_core;  /* |z|^2 < HK_Z2: 4-point Gauss-Hermite (outer ring), 6-point, trapezoid + pole term innermost */
    int64_t n_evals_gh6;   /* of n_evals_core: the 6-point ring (HK_Z3 <= |z|^2 < HK_Z4 at small y; see HK_Z4 for its dependence on y) */
    int64_t n_evals_trap;  /* of n_evals_core: |z|^2 < HK_Z3 (21 when y >= 1) and y < 3 (trapezoid, or 10-point Gauss-Hermite when y >= 1.8) */
    int64_t n_units_far;   /* (tile, line-chunk) work units run by the far kernel */
    int64_t n_units_mid;   /* ... by the mid kernel */
    int64_t n_units_near;  /* ... by the near/edge kernel */
    int64_t n_pairs_far;   /* (line, bin) pairs the far kernel evaluated (mask-free Lorentzian) */
    int64_t n_pairs_mid;   /* (line, bin) pairs the mid kernel evaluated (mask-free two-term asymptotic) */
    int64_t n_pairs_near;  /* (line, bin) slots the generic near kernel walked (masked; includes bins outside extents) */
    int64_t n_units_node;  /* ... by the node kernel */
    int64_t n_units_edge;  /* ... by the edge kernel */
    int64_t n_units_centre; /* ... by the centre kernel */
    int64_t n_pairs_edge;  /* (line, bin) slots the edge kernel walked (masked two-term; includes bins outside extents) */
    int64_t n_pairs_centre; /* (line, bin) slots the centre kernel walked (two-term outside the core, core evaluators inside) */
    int64_t n_pairs_node;  /* (line, tile) pairs evaluated at the tile's HK_NODES Chebyshev nodes (two-term asymptotic) */
    int64_t n_bins_node;   /* (line, bin) pairs those node evaluations stand for */
    int64_t n_evals_gh10;  /* of n_evals_trap: lines with y >= 1.8, evaluated by the 10-point Gauss-Hermite rule */
    int64_t n_pairs_edge_node; /* (line, extent end) pairs evaluated at the nodes of their edge tile (per-bin accumulators) */
    int64_t n_launches;    /* kernels of this library launched by the last hk_compute (CUB passes excluded) */
    int64_t n_plinth_illcond; /* plinth removal: lines with V(cut) > V(0) / HK_PLINTH_RATIO, whose difference V - V(cut) is
                                 ill-conditioned in fp32 (see hk_set_plinth: 0 means the subtracted result meets the tolerance) */
    int64_t n_evals_gh10_row; /* of n_evals_gh10: evaluated by the row kernel (lines at least 0.85 bins wide per 64 bins of tile); the rest by the lane kernel */
    int64_t n_pairs_node_eval; /* (line, tile) pairs the node kernel evaluated; equals n_pairs_node (checked by the tests) */
    int64_t n_pairs_node_far; /* of n_pairs_node: |z|^2 >= HK_Z1 on the whole tile, evaluated with one asymptotic term */
    int64_t n_unsorted;    /* adjacent pairs of the input list out of centre-bin order (0: the list arrived sorted and the
                              radix sort was skipped on the device) */
    int64_t n_evals_core_nodes; /* of n_evals_core: bins of tiles the node hierarchy handles (hk_set_core_nodes): covered by the
                                   interpolant of the tile's node values, not evaluated one by one */
    int64_t n_pairs_node_core; /* of n_pairs_node: the tile may hold bins with |z|^2 < HK_Z2 (a separated tile of the core, outside
                                  the inner region): evaluated at the nodes with the 4-point Gauss-Hermite form */
    int32_t scale_exp;     /* per-launch power-of-two scale applied to line strengths */
    int32_t sort_bits;     /* radix-sort key width used */
    int32_t bins_per_lane; /* tile geometry used: a level-0 tile is 32 x this many bins */
    int32_t n_levels;      /* levels of the node hierarchy used (0: direct evaluation only) */
    int32_t single_pass;   /* 1: the records of the last compute were written by the single-pass preprocess (hk_set_single_pass) */
    int32_t reserved0;
} hk_stats;

/* Phases of one hk_compute, timed with CUDA events on the caller's stream. */
enum { HK_PH_PREPROCESS = 0, HK_PH_SORT = 1, HK_PH_RANGES = 2, HK_PH_NODE = 3, HK_PH_FAR = 4, HK_PH_MID = 5, HK_PH_EDGE = 6,
       HK_PH_CENTRE = 7 /* line centres, row kernel */, HK_PH_LANE = 8 /* line centres, innermost bins */, HK_PH_NEAR = 9,
       HK_PH_DOWN = 10, HK_PH_COUNT = 11 };

/* Region thresholds on |z|^2 = x^2 + y^2 used by the fp32 evaluator. */
#define HK_Z1 90000.0f /* |z| >= 300: one asymptotic term, relative error <= 1.7e-5 */
#define HK_Z2 625.0f   /* |z| >= 25 : two asymptotic terms, relative error <= 1.0e-5 */
#define HK_Z4 49.0f    /* 7 <= |z| < 25: 4-point Gauss-Hermite rational form, <= 3e-6; below: 6-point.  The rings shrink as y grows
                          (the pole moves away from the real axis): 4 points from |z|^2 >= 36 for y >= 1.5, >= 30.25 for y >= 3, and
                          on the whole core for y >= 4.5; 6 points on the whole core for y >= 3 (hk_device.cuh: z4_for, z3_for) */
#define HK_Z3 30.25f   /* |z| < 5.5 (|z|^2 < 50 when y < 1e-3, < 21 when y >= 1) and y < 3: trapezoid rule + pole term, <= 2e-6; 10-point Gauss-Hermite when y >= 1.8, <= 9e-6 */
#ifndef HK_NODES
#define HK_NODES 12    /* Chebyshev nodes per tile of the separated-tile evaluation; 8, 10 or 12 */
#endif
#define HK_NODE_SEP (HK_NODES == 8 ? 4.0 : HK_NODES == 10 ? 2.5 : 2.0) /* default separation, tile half-widths: interpolation error <= 6e-6 */
#define HK_NODE_SEP_PLINTH (HK_NODE_SEP + 1.0) /* smallest separation used with plinth removal (hk_set_plinth): ~3e-8 of the
                                                  unsubtracted value, which the subtraction amplifies towards the extent ends */

/* Grid: bin i is the POINT nu_i = numin + i*dnu (R8, R9).  HK_EINVAL if dnu <= 0,
 * numax <= numin, a non-finite argument, N < 1 or N too large. */
int hk_create(double numin, double numax, double dnu, hk_ctx** out);
int hk_destroy(hk_ctx* ctx);
int64_t hk_grid_size(const hk_ctx* ctx);

/* T in K, P in atm, molecular/atomic mass in amu, partition function Q(T) as a
 * scalar (Eq. 10 is evaluated by the caller, L234).  HK_EINVAL unless T, mass, Q > 0,
 * P >= 0, all finite. */
int hk_set_conditions(hk_ctx* ctx, double T_K, double P_atm, double mass_amu, double Q);

/* Line profile (section 2.1: Voigt, and "sometimes pure Doppler and Lorentzian profiles are also used"), unit area:
 *   HK_PROFILE_VOIGT   Re w(x + i y)/(alpha_D sqrt(pi))                      (default)
 *   HK_PROFILE_LORENTZ Gamma_L/(pi ((nu - nu0)^2 + Gamma_L^2))
 *   HK_PROFILE_DOPPLER exp(-((nu - nu0)/alpha_D)^2)/(alpha_D sqrt(pi))
 *   HK_PROFILE_BINNED_GAUSSIAN  the "binned Gaussian integrated cross section" of ExoCross (L47): the Doppler profile
 *                      averaged over each bin, (1/(2 dnu)) [erf((nu_i + dnu/2 - nu0)/alpha_D) - erf((nu_i - dnu/2 - nu0)/alpha_D)]
 *                      (PAPER.md names it and prints no formula: DESIGN.md R26); conserves sum_i V_i dnu = 1 at any resolution
 * Dynamic range of one launch (every profile): the fp32 evaluation carries ONE power-of-two scale per launch, set from
 * the largest line amplitude of the list; a term more than ~166 binades (1e-50; Gaussian profiles: 226 binades, 1e-68)
 * below the largest amplitude is flushed to zero.  Such terms are below every tolerance unless the WHOLE spectrum
 * is -- a pure Gaussian is followed down to exp(-157) of its peak, where that range ends.
 * HK_EINVAL for any other value. */
#define HK_PROFILE_VOIGT 0
#define HK_PROFILE_LORENTZ 1
#define HK_PROFILE_DOPPLER 2
#define HK_PROFILE_BINNED_GAUSSIAN 3
int hk_set_profile(hk_ctx* ctx, int profile);

/* Cutting length (L239: "a fixed cutting length, a fraction of the Doppler half-width, or a fraction of the Lorentzian
 * half-width"): what the cut_cm argument of the compute entry points means.
 *   HK_CUT_FIXED    cut_cm is the cutting length in cm^-1, the same for every line        (default)
 *   HK_CUT_LORENTZ  the cutting length of a line is cut_cm x its Gamma_L
 *   HK_CUT_DOPPLER  the cutting length of a line is cut_cm x its Gamma_D = alpha_D sqrt(ln 2)
 * A line of zero half-width has no extent.  cut_cm <= 0 or +inf is uncut in every mode.  In the width-relative modes
 * a compute reads the range of cutting lengths back (ONE host synchronisation per call) and runs one pass per class
 * [c, 2c) of cutting length, so the call is synchronous up to its last pass; hk_compute_host does not support them.
 * hk_get_stats afterwards: n_evals / n_skipped / n_off_grid are totals, the rest describes the last pass. */
#define HK_CUT_FIXED 0
#define HK_CUT_LORENTZ 1
#define HK_CUT_DOPPLER 2
int hk_set_cut_mode(hk_ctx* ctx, int mode);

/* Plinth removal (section 2.1.1): on != 0 subtracts from every bin of a line's extent that line's own value
 * at the cutting length position, S V(nu0 +- cut) (needed with continua that already hold the plinths, e.g. CKD).
 * Off by default; no effect on uncut computations.  Changes hk_workspace_bytes (+ 8 B per bin): set it before the
 * workspace is sized.  Applies to hk_compute, hk_accumulate, hk_compute_batch and hk_compute_host.
 * Accuracy contract: S (V - V(cut)) is a difference of two fp32 evaluations, each good to a few 1e-7 (rounding) to
 * 1e-6 (inside the core) of ITSELF.  While every line's value at its cutting length is small against its peak,
 * V(cut) <= V(0) / HK_PLINTH_RATIO -- the normal use: a cut of many half-widths -- the SUBTRACTED opacity meets the
 * tolerance of the library (1e-4 per bin relative to the result, 1e-8 max(k) below that: the bins next to the extent's
 * ends, where the difference vanishes, fall under the absolute branch) up to the ROUNDING of its two terms, 2^-22
 * (HK_PLINTH_ROUNDING) of the opacity before removal -- which shows only where an isolated line's subtracted value is
 * below ~0.2 % of its unsubtracted one and still above 1e-8 max(k), the last bins before an extent end.  Separated tiles
 * are evaluated at HK_NODE_SEP_PLINTH half-widths (interpolation error 3e-8 instead of 6e-6 of the unsubtracted value:
 * it would not cancel against the directly evaluated plinth).  A line that does not is counted in
 * hk_stats.n_plinth_illcond (cut inside the line's core, or shorter than ~23 Lorentz half-widths); in the bins such
 * lines dominate the result is then good to 1e-4 of the opacity BEFORE removal only -- no fp32 evaluation can do better
 * -- and a caller who needs more must use a longer cut. */
#define HK_PLINTH_RATIO 512.0
#define HK_PLINTH_ROUNDING 2.384185791015625e-07 /* 2^-22 */
int hk_set_plinth(hk_ctx* ctx, int on);

/* Device scratch the caller must provide for hk_compute with up to n_lines lines. */
size_t hk_workspace_bytes(const hk_ctx* ctx, int64_t n_lines);
int hk_set_workspace(hk_ctx* ctx, void* dev_ptr, size_t bytes);

/* Reproducibility: lines of one centre bin keep no fixed order among themselves (counting sort; the single-pass
 * preprocess keeps the caller's), fp32 partial sums of up to 128 terms follow that order, and bins receive them through
 * fp64 atomic adds whose order is not fixed either: two runs of the same call agree to the rounding of those sums
 * (a few 1e-7 of the local k at most, usually far less), not bit for bit (the paper notes the same of its summation
 * order, L666).  Integer outputs (extents, counts) are exact and reproducible.
 *
 * Enqueue the whole hot path on `stream` (a cudaStream_t passed as void*; NULL is
 * the legacy default stream): preprocess -> sort by centre bin -> tile ranges -> node, far, mid, extent-end,
 * centre and near accumulation kernels -> interpolation of the node sums (-> plinth removal) -> k in out_k_dev.
 * out_k_dev (N doubles) is OVERWRITTEN.  cut_cm > 0 and finite: cutting length from the centre (cm^-1, or a
 * multiple of the line's half-width: hk_set_cut_mode), inclusive integer extent (R7); cut_cm <= 0 or +inf: uncut.
 * Lines need not be sorted.  n_lines == 0 is valid (k = 0).  Returns after enqueueing, without synchronising
 * (except in the width-relative cut modes, see hk_set_cut_mode); every buffer must stay alive until the stream
 * drains.  The profile, plinth and cut-mode settings of the context apply. */
int hk_compute(hk_ctx* ctx, const hk_lines* lines, int64_t n_lines, double cut_cm,
               double* out_k_dev, void* stream);

/* hk_compute for callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): the workspace is a static device array inside the library, HK_STATIC_WS_BYTES
 * (32 MiB) that every GPU which loads libhk.so holds until the process exits.  The call allocates nothing and frees
 * nothing (no cudaMalloc / cudaFree / allocating library routine; the temporary storage of the CUB scans and sorts lies
 * in the array too), needs no hk_set_workspace, and leaves a workspace bound with hk_set_workspace as it was.  Same
 * definition, arguments, asynchrony and results as hk_compute (lines and out_k_dev are the caller's device buffers),
 * for problems with hk_workspace_bytes(ctx, n_lines) <= HK_STATIC_WS_BYTES: about 1e5 lines on 5e4 bins, or 2e5 lines
 * on 1e4 bins (~140 B per line + ~200 B per bin); anything larger returns HK_ENOSPC before touching the GPU.  Fixed
 * cutting length or none only (HK_ESTATE in the width-relative cut modes).  The first call on a device resolves the
 * array's device address (cudaGetSymbolAddress; HK_ECUDA with hk_last_cuda_error if that fails).
 * ONE array per device, shared by every context and every call: it holds the last call's contents (what must start at
 * zero is cleared on `stream` by the call itself), so two calls whose GPU work OVERLAPS -- different streams, different
 * contexts, different host threads -- race; order them on one stream or with events.  hk_get_stats / hk_get_extents /
 * hk_get_phase_ms afterwards describe this call as long as no later hk_compute_static has run. */
#define HK_STATIC_WS_BYTES (32u << 20)
int hk_compute_static(hk_ctx* ctx, const hk_lines* lines, int64_t n_lines, double cut_cm,
                      double* out_k_dev, void* stream);

/* Same as hk_compute but ADDS into out_k_dev instead of overwriting it (line lists that
 * arrive in blocks, L187: the sum over lines is order-independent, R16). */
int hk_accumulate(hk_ctx* ctx, const hk_lines* lines, int64_t n_lines, double cut_cm,
                  double* out_k_dev, void* stream);

/* Many (T, P, Q) points on one resident line list in one call (the paper's "multiple pressure points per run",
 * L361, L733, Table 8: the lines stay on the GPU across the points).  T_K, P_atm, Q: HOST arrays of n_cond
 * values (the mass of hk_set_conditions applies to all; hk_set_conditions must have been called and its T, P, Q are
 * left untouched).  out_k_dev: DEVICE array of n_cond x N doubles, row c = k(nu) at condition c, OVERWRITTEN.
 * Every point is the full definition of hk_compute at that condition; what is shared is what does not depend on the
 * condition: the order of the lines by centre bin (one sort for the batch) and the workspace -- and, between consecutive
 * points that differ in PRESSURE only (same T and Q: the paper's pressure sweeps), everything but the Lorentz widths:
 * strengths, Doppler widths, centre bins, extents, tile and node ranges are kept and one streaming pass rewrites
 * (Gamma_L/dnu)^2 and what follows from it in the sorted records (plain Voigt profile, fixed cut or none, no plinth
 * removal; otherwise the point runs the full preprocess on the shared order).  Order the points by temperature.  All conditions are
 * validated before anything is enqueued (HK_EINVAL as hk_set_conditions).  n_cond == 0 is valid.  Asynchronous like
 * hk_compute.  hk_get_stats afterwards describes the LAST condition, n_launches the whole batch. */
int hk_compute_batch(hk_ctx* ctx, const hk_lines* lines, int64_t n_lines, double cut_cm, int32_t n_cond,
                     const double* T_K, const double* P_atm, const double* Q, double* out_k_dev, void* stream);

/* A wavenumber axis made of bands of different resolution (L218: "it is possible to use a different wavenumber
 * resolution for different bands"): one context per band (its own numin, numax, dnu, conditions and workspace; the
 * workspaces may be one buffer if the bands run on one stream), one output array per band; every band is the full
 * definition of hk_compute on its own grid, so a line near a band edge contributes to both bands through its clamped
 * extent.  ctxs, out_k_dev: HOST arrays of n_bands pointers.  All bands are checked before anything is enqueued. */
int hk_compute_bands(hk_ctx* const* ctxs, int32_t n_bands, const hk_lines* lines, int64_t n_lines, double cut_cm,
                     double* const* out_k_dev, void* stream);

/* ---- HITRAN-style inputs (Table 3-4: nu, E_L, A, delta, gamma_air, gamma_self, n per line) -----------
 * Nine SoA DEVICE arrays of n_lines elements, read-only: eight fp64 and the int32 isotopologue index of each line
 * into the table given to hk_set_conditions_hitran (the species parameter file's isotopologue list, L371-373). */
typedef struct {
    const double* nu0;        /* tabulated line centre, cm^-1 */
    const double* A;          /* Einstein A, s^-1 */
    const double* g_up;       /* upper-state degeneracy */
    const double* E_low;      /* lower-state energy, cm^-1 */
    const double* gamma_air;  /* air-broadening coefficient at T_ref, cm^-1/atm */
    const double* gamma_self; /* self-broadening coefficient at T_ref, cm^-1/atm */
    const double* n_exp;      /* temperature exponent n */
    const double* delta;      /* pressure shift, cm^-1/atm */
    const int32_t* iso;       /* isotopologue index, 0 .. n_iso-1 */
} hk_lines_hitran;

/* Conditions for HITRAN-style lists:
 *   Gamma_L = A/(4 pi c) + (T/T_ref)^-n [gamma_air (P - P_self)/P_ref + gamma_self P_self/P_ref]        (Eq. 4)
 *   centre  = nu0 + delta P        (pressure shift, L238; the reason the paper re-sorts the lines)
 *   alpha_D = (nu0/c) sqrt(2 k_B T/m_iso);  S = abundance_iso x Eq. 9 with m_iso and Q_iso(T)
 * The profile and the integer extent are centred on the SHIFTED centre; S and alpha_D use the tabulated nu0
 * (R23, R24).  mass_amu, Q, abundance: HOST arrays of n_iso (1..16) entries.  HK_EINVAL unless T > 0,
 * 0 <= P_self <= P, masses and Q > 0, abundances >= 0, all finite.  A line whose iso is outside the table contributes
 * nothing (counted in n_skipped).  Also sets the ExoMol-style conditions to (T, P, mass[0], Q[0]). */
int hk_set_conditions_hitran(hk_ctx* ctx, double T_K, double P_atm, double P_self_atm, int32_t n_iso,
                             const double* mass_amu, const double* Q, const double* abundance);

/* hk_compute for a HITRAN-style list: same hot path after the per-line preprocessing; workspace as hk_compute
 * (hk_workspace_bytes).  HK_ESTATE before hk_set_conditions_hitran. */
int hk_compute_hitran(hk_ctx* ctx, const hk_lines_hitran* lines, int64_t n_lines, double cut_cm, double* out_k_dev,
                      void* stream);

/* Per-line parameters and integer extents (of the shifted centre, for cut_cm) as the preprocess kernel computes
 * them: parity of step a1 for HITRAN-style lists.  DEVICE arrays of n_lines, any may be NULL.  Synchronises. */
int hk_get_line_params_hitran(hk_ctx* ctx, const hk_lines_hitran* lines, int64_t n_lines, double cut_cm, double* S_dev,
                              double* gammaL_dev, double* alphaD_dev, int32_t* ilo_dev, int32_t* ihi_dev,
                              int32_t* jc_dev, void* stream);

/* Host-buffer entry (the paper's block pipeline, L183-189, Fig. 6): the six line
 * arrays and out_k are HOST pointers (pinned memory gives asynchronous copies; pageable
 * works, slower).  The list is cut into blocks of block_lines lines (<= 0: default 2^25);
 * block b+1 is copied host->device on an internal copy stream while block b runs
 * hk_accumulate on `stream`; k is copied back once at the end.  Device scratch comes
 * from the workspace set with hk_set_workspace, which must hold
 * hk_workspace_bytes_host(ctx, n_lines, block_lines).  SYNCHRONOUS: returns when
 * out_k_host holds the result.  hk_get_stats afterwards reports the LAST block only,
 * except n_lines / n_evals / n_skipped, which are totals. */
size_t hk_workspace_bytes_host(const hk_ctx* ctx, int64_t n_lines, int64_t block_lines);
int hk_compute_host(hk_ctx* ctx, const hk_lines* host_lines, int64_t n_lines, double cut_cm,
                    double* out_k_host, int64_t block_lines, void* stream);

/* Integer extents of the lines of the LAST compute, in the caller's line order
 * (int32 DEVICE arrays of n_lines; skipped / off-grid lines get ilo = 0, ihi = -1,
 * jc as computed (0 for skipped)).  Any pointer may be NULL.  Synchronises.
 * When n_lines equals that of the last compute and it ran as one pass (hk_compute / hk_accumulate / hk_compute_hitran
 * with a fixed cut or none, a single-block hk_compute_host) the values are the ones that compute WROTE -- read from its
 * per-line records, shifted centres and all -- and `lines` is not read (may be NULL).  Otherwise (width-relative
 * cutting lengths, several blocks: the record buffer held one pass at a time) they are recomputed from `lines` with
 * the conditions, cut and cut mode of the last compute; HK_ESTATE in that case after hk_compute_hitran (use
 * hk_get_line_params_hitran). */
int hk_get_extents(hk_ctx* ctx, const hk_lines* lines, int64_t n_lines, int32_t* ilo_dev,
                   int32_t* ihi_dev, int32_t* jc_dev, void* stream);

/* Per-line fp64 parameters as the preprocess kernel computes them (S, Gamma_L,
 * alpha_D; zeros for skipped lines): parity of step a1.  DEVICE arrays, may be NULL. */
int hk_get_line_params(hk_ctx* ctx, const hk_lines* lines, int64_t n_lines, double* S_dev,
                       double* gammaL_dev, double* alphaD_dev, void* stream);

/* Counts of the last hk_compute.  Synchronises the stream it ran on. */
int hk_get_stats(hk_ctx* ctx, hk_stats* host_out);

/* Milliseconds per phase (HK_PH_*) of the last hk_compute / hk_accumulate, from CUDA
 * events recorded on its stream between the phases.  out_ms: HOST array of
 * HK_PH_COUNT floats.  Synchronises. */
int hk_get_phase_ms(hk_ctx* ctx, float* out_ms);

/* FP32 issue-rate probes for the roofline denominator ("measure an FFMA peak and the clock actually
 * held"): 16 independent register-resident chains per thread on every SM (4 CTAs x 512 threads per SM), one
 * instruction kind per launch:
 *   kind 0  FFMA2 (fma.rn.f32x2), three distinct register operands      3  FADD2 (add.rn.f32x2)
 *        1  scalar FFMA, three register operands                        4  FMUL2 (mul.rn.f32x2)
 *        2  FFMA2 with scalar multiplier and addend (broadcast form)    5  MUFU.RCP (rcp.approx.ftz.f32)
 * *lane_ops_per_s (HOST): fp32 lane operations per second (an FMA is one operation: x2 for FLOP/s);
 * *sm_clock_mhz (HOST, may be NULL): SM cycles / nanoseconds measured INSIDE the kernel (clock64 / globaltimer), i.e.
 * the SM clock actually held during the probe; *ms_out (may be NULL): kernel time.  Run it with iters large enough
 * for >= 200 ms when the point is the sustained clock.  Synchronises.
 * hk_probe_fp32_peak(packed, ...) = 2 x the kind-0 (packed != 0) or kind-1 rate, in FLOP/s. */
int hk_probe_fp32_ops(int kind, int iters, double* lane_ops_per_s, double* sm_clock_mhz, float* ms_out, void* stream);
int hk_probe_fp32_peak(int packed, int iters, double* flops_out, float* ms_out, void* stream);

/* Accuracy probe for the shipped fp32 evaluator (the counterpart of the paper's
 * Fig. 4): out[i] = Re w(x[i] + i y[i]) exactly as the accumulation
 * kernels evaluate it (region chosen by |z|^2 with alpha_D = 1 bin).  DEVICE fp32
 * arrays of n.  region_out (optional, int32): 0 far, 1 mid, 2 Gauss-Hermite 4, 3 Gauss-Hermite 6, 4 trapezoid,
 * 5 Gauss-Hermite 10 (|z|^2 < HK_Z3 and y >= 1.8). */
int hk_eval_voigt_f32(const float* x_dev, const float* y_dev, int64_t n, float* out_dev,
                      int32_t* region_out_dev, void* stream);

/* Knobs for tests and sweeps.  mode 0: the default split (separated tiles at Chebyshev nodes, the rest
 * directly); mode 3: direct evaluation of every (line, bin) pair with the far / mid / near split;
 * mode 1: every pair through the near/edge kernel; mode 2: far pairs through the mid (two-term) kernel
 * (modes 1-3 do not use the node hierarchy).
 * hk_set_node_separation: a (line, tile) pair is evaluated at nodes when the line centre is at least
 * `sep` tile half-widths from the tile centre (default 4; 0 disables the hierarchy; HK_EINVAL for 0 < sep < 3, where the
 * degree-7 interpolant leaves the error budget of DESIGN.md section 5, and for sep > 64).
 * hk_set_tile_bins: bins per lane 2, 4 or 8 (a warp owns 32x, a CTA 256x); 0 = chosen from
 * the cut (include/hk.h hk_stats.bins_per_lane reports the choice). */
int hk_set_debug_mode(hk_ctx* ctx, int mode);
int hk_set_tile_bins(hk_ctx* ctx, int bins_per_lane);
int hk_set_node_separation(hk_ctx* ctx, double sep);
/* on (default): tiles an extent covers only in part, when separated from the line, are evaluated at the tile's nodes
 * into per-bin accumulators (128 B per bin of workspace, used while that is <= 1 GiB); off: masked direct evaluation. */
int hk_set_edge_nodes(hk_ctx* ctx, int on);
/* 0 (default): the line-stationary node kernel (node_lines_kernel); 1: the entry-stationary one it replaced (node_kernel).
 * Both evaluate exactly the (line, tile) pairs node_range_kernel lists, with the same arithmetic per pair: a cross-check. */
int hk_set_node_kernel(hk_ctx* ctx, int entry_stationary);
/* The core at nodes (default on).  The Voigt profile is smooth enough for the 12 Chebyshev nodes of a tile wherever the
 * tile is separated from the line (hk_set_node_separation) and lies outside the line's INNER region -- not only in the
 * asymptotic wings: with |z|^2 >= 49 on all of the tile the interpolation error stays below 1.3e-5 (measured against the
 * oracle's profile, tests/test_nodes.py).  on: such tiles of the core go through the node hierarchy, their node values
 * from the 4-point Gauss-Hermite form (plain Voigt profile, fixed cut or none, outside hk_compute_batch); off: the
 * hierarchy takes tiles with |z|^2 >= HK_Z2 only and the centre kernels evaluate every bin of the core directly. */
int hk_set_core_nodes(hk_ctx* ctx, int on);
/* Single-pass preprocess (default on).  Line lists are stored in wavenumber order (L216-218) and a caller's conditions
 * move little between calls, so every compute leaves a 16-byte HINT in the workspace: "the list arrived in centre-bin
 * order with every line valid and on the grid" and the exponent of its launch scale.  The next hk_compute / hk_accumulate
 * / hk_compute_hitran on that workspace (fixed cut, no plinth, not the binned Gaussian) then writes the sorted fp32
 * records in ONE pass over the lines, and checks both assumptions on the device while it does: a line without a key, a
 * pair out of order, or a hinted scale more than 8 binades from the one this call's own maxima ask for, and the call
 * runs the ordinary two passes (per-line parameters, then counting sort) after all -- same launches either way, nothing
 * decided on the host.  Same fp64 and fp32 arithmetic per line on both paths; the launch scale is a power of two, so
 * the result does not depend on which path ran (beyond fp32 under/overflow 2^100 away from the largest amplitude).
 * The first compute on a workspace, an unsorted list and a list with lines off the grid always take the two passes.
 * hk_stats.single_pass says which path the last compute took.  off: always two passes. */
int hk_set_single_pass(hk_ctx* ctx, int on);

int hk_last_cuda_error(const hk_ctx* ctx);
const char* hk_strerror(int status);

#ifdef __cplusplus
}
#endif
#endif /* HK_H */
