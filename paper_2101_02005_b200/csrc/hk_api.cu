// hk_api.cu -- host side of the C ABI in include/hk.h: argument checks, workspace
// layout, and the enqueue of the whole hot path on the caller's stream.  No host
// synchronisation inside hk_compute: launch shapes do not depend on device results
// (persistent grids pull work units from a device-computed list).
#include <cub/device/device_radix_sort.cuh>
#include <cub/device/device_scan.cuh>

#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>
#include <type_traits>

#include "hk_accumulate.cuh"

using namespace hk;

struct hk_ctx {
    double numin, numax, dnu;
    int64_t N;
    bool have_cond;
    double T, P_atm, mass_amu, Q;
    void* ws;
    size_t ws_bytes;
    int cuda_err;
    int debug_mode;
    int force_kb;
    double node_sep;
    int edge_nodes;
    int node_entry_stationary;   // test knob: the entry-stationary node kernel instead of the line-stationary one
    int plinth;
    int profile;
    int cut_mode;
    // HITRAN-style conditions (hk_set_conditions_hitran)
    bool have_hitran;
    double P_self;
    int32_t n_iso;
    double iso_mass[kMaxIso], iso_Q[kMaxIso], iso_ab[kMaxIso];
    int n_sm;
    // last compute
    bool have_run;
    int64_t last_n;
    double last_cut;
    cudaStream_t last_stream;
    int32_t last_sort_bits, last_kb, last_levels;
    int64_t last_launches;
    DevStats* d_stats;
    // sorted records of the last pass (for the on-demand region counts and hk_get_extents) with the sort's permutation
    const float4 *last_recA, *last_recB, *last_recN;
    const int32_t* last_idx;
    int core_nodes;              // 1 (default): separated tiles of the core outside the inner region go to the node hierarchy
    int single_pass;             // 1 (default): a list the previous compute found sorted is preprocessed in one pass
    bool hint_ready;             // the DevHint of the bound workspace has been initialised
    bool in_batch;               // inside hk_compute_batch: tile ranges may serve later conditions with other widths
    int last_profile;
    Params last_p;               // the launch constants and node levels of the last pass (for the on-demand counts)
    Levels last_lv;
    bool regions_done;
    // totals over the blocks of the last hk_compute_host (0 after a plain hk_compute)
    bool host_totals;            // the counts of the last call are totals kept on the device (d_totals)
    int64_t tot_lines;
    DevTotals* d_totals;
    bool last_multi;             // the last call ran several passes / blocks: recU holds the last one only
    bool last_hitran;
    // phase events (recorded on the caller's stream) and the host-pipeline resources
    cudaEvent_t ev[HK_PH_COUNT + 1];
    cudaStream_t copy_stream;
    cudaEvent_t ev_h2d[2], ev_done[2];
};

namespace {

inline size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

struct Layout {
    size_t stats, totals, hint, keys_in, keys_out, idx_in, idx_out, recU, flo, recA, recB, recN, recC, tr, nr, node_acc, edge_acc, plinth_acc, counts, prefix, cub;
    size_t edge_acc_bytes;   // 0: grid too large for the per-bin edge accumulators (direct edge kernel only)
    size_t cub_bytes, total;
    int32_t n_ct;        // level-0 tiles of the smallest geometry
    int32_t n_entries;   // upper bound on (level, tile) entries of the node hierarchy
    int32_t n_counts;    // work-unit counts: 6 n_ct (far, mid, edge, centre, near, lane) + n_entries (node) + 1
};

bool is_uncut(double cut) { return !(cut > 0.0 && std::isfinite(cut)); }

size_t cub_temp_bytes(int64_t n, int32_t n_ct, int64_t n_bins)
{
    size_t b1 = 0, b2 = 0, b3 = 0;
    cub::DeviceScan::InclusiveSum(nullptr, b3, (const double*)nullptr, (double*)nullptr, (int)(n_bins + 1), (cudaStream_t)0);
    cub::DeviceRadixSort::SortPairs(nullptr, b1, (const int32_t*)nullptr, (int32_t*)nullptr, (const int32_t*)nullptr,
                                    (int32_t*)nullptr, (int)n, 0, 32, (cudaStream_t)0);
    cub::DeviceScan::ExclusiveSum(nullptr, b2, (const int32_t*)nullptr, (int32_t*)nullptr, (int)n_ct,
                                  (cudaStream_t)0);
    if (b3 > b1) b1 = b3;
    return b1 > b2 ? b1 : b2;
}

constexpr int kMinKB = 2;     // smallest tile geometry: the workspace is sized for it

// bins per lane from the half-extent in bins: wide extents amortise the per-line work over more
// bins; narrow ones need small warp tiles so that most (line, tile) pairs are interior.
int pick_kb(const hk_ctx* c, double cut)
{
    if (c->force_kb) return c->force_kb;
    // measured (profiles/): with the node hierarchy taking every separated tile, small level-0 tiles win whenever
    // there is a cut (fewer direct near-field pairs, smaller edge tiles); uncut lists are sparse and favour wide tiles
    return is_uncut(cut) ? 8 : 2;
}

Layout make_layout(const hk_ctx* c, int64_t n)
{
    Layout L;
    L.n_ct = (int32_t)((c->N + 32 * kMinKB - 1) / (32 * kMinKB));
    L.n_entries = 2 * L.n_ct + kMaxLevels;
    L.n_counts = 6 * L.n_ct + L.n_entries + 1;
    size_t nn = (size_t)(n > 0 ? n : 1);
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off += align_up(bytes); return o; };
    L.stats = take(sizeof(DevStats));
    L.totals = take(sizeof(DevTotals));      // (fixed offset: survives the per-block layouts of hk_compute_host)
    L.hint = take(sizeof(DevHint));          // (fixed offset too: carried from one compute to the next)
    L.keys_in = take(nn * 4);
    L.keys_out = take(nn * 4);
    L.idx_in = take(nn * 4);
    L.idx_out = take(nn * 4);
    L.recU = take(nn * sizeof(RecU));
    L.flo = take(c->profile == HK_PROFILE_BINNED_GAUSSIAN ? nn * 4 : 0);   // low part of the sub-bin offset (R26)
    L.recA = take(nn * 16);
    L.recB = take(nn * 16);
    L.recN = take(nn * 16);
    L.recC = take(nn * 16);
    L.tr = take((size_t)L.n_ct * sizeof(TileRange));
    L.nr = take((size_t)L.n_entries * sizeof(NodeRange));
    L.node_acc = take((size_t)L.n_entries * kP * sizeof(double));
    // per-bin node sums of the extent ends: [2][N][kP] fp64 = 128 B per bin, used up to 1 GiB
    L.edge_acc_bytes = (size_t)2 * (size_t)c->N * kP * sizeof(double);
    if (L.edge_acc_bytes > ((size_t)1 << 30)) L.edge_acc_bytes = 0;
    L.edge_acc = take(L.edge_acc_bytes);
    L.plinth_acc = take(c->plinth ? (size_t)(c->N + 1) * sizeof(double) : 0);
    L.counts = take((size_t)L.n_counts * 4);
    L.prefix = take((size_t)L.n_counts * 4);
    L.cub_bytes = cub_temp_bytes((int64_t)nn, L.n_counts, c->N);
    L.cub = take(L.cub_bytes);
    L.total = off;
    return L;
}

int fail_cuda(hk_ctx* c, cudaError_t e)
{
    if (c) c->cuda_err = (int)e;
    return HK_ECUDA;
}

#define HK_CUDA(call)                                   \
    do {                                                \
        cudaError_t e__ = (call);                       \
        if (e__ != cudaSuccess) return fail_cuda(ctx, e__); \
    } while (0)

// Fill the per-launch constants (step a0).
struct CutClass {
    double lo, hi;          // lines with lo <= cutting length < hi belong to the pass
    double bound_lo, bound_hi;   // smallest / largest cutting length that can occur in it (cm^-1)
    bool first;
};

Params make_params(const hk_ctx* c, double cut, int32_t chunk, bool hitran = false, const CutClass* cls = nullptr)
{
    Params p;
    std::memset(&p, 0, sizeof(p));
    p.numin = c->numin;
    p.dnu = c->dnu;
    p.inv_dnu = 1.0 / c->dnu;
    p.N = c->N;
    const double m = c->mass_amu / kNA;                        // grams (L83)
    p.c2_over_T = kH * kC / kKB / c->T;
    p.tfac = kTref / c->T;
    p.ln_tfac = std::log(p.tfac);
    p.P_atm = c->P_atm;
    p.beta = std::sqrt(2.0 * kKB * c->T / m) / kC;
    p.sfac = 1.0 / (8.0 * kPi * kC * m * c->Q);
    p.cKfac = p.sfac / (p.beta * std::sqrt(kPi));
    p.inv4pic = 1.0 / (4.0 * kPi * kC);
    if (hitran) {
        // per isotopologue: Doppler factor and abundance / (8 pi c m Q); the tile bounds use the widest Doppler factor
        p.P_self = c->P_self;
        p.n_iso = c->n_iso;
        p.beta = 0.0;
        for (int j = 0; j < c->n_iso; ++j) {
            const double mj = c->iso_mass[j] / kNA;
            p.beta_iso[j] = std::sqrt(2.0 * kKB * c->T / mj) / kC;
            p.sfac_iso[j] = c->iso_ab[j] / (8.0 * kPi * kC * mj * c->iso_Q[j]);
            p.cKfac_iso[j] = p.sfac_iso[j] / (p.beta_iso[j] * std::sqrt(kPi));
            if (p.beta_iso[j] > p.beta) p.beta = p.beta_iso[j];
        }
    }
    p.uncut = is_uncut(cut) ? 1 : 0;
    p.cut = p.uncut ? 0.0 : cut;
    p.cut_mode = p.uncut ? 0 : c->cut_mode;
    p.cut_factor = cut;
    p.cls_lo = 0.0;
    p.cls_hi = INFINITY;
    p.count_invalid = 1;
    double cb = p.uncut ? 0.0 : cut / c->dnu;
    double cb_lo = cb, cb_hi = cb;                 // bounds of the cutting length in bins: one value unless width-relative
    if (p.cut_mode != 0 && cls) {
        p.cls_lo = cls->lo; p.cls_hi = cls->hi; p.count_invalid = cls->first ? 1 : 0;
        cb_lo = cls->bound_lo / c->dnu; cb_hi = cls->bound_hi / c->dnu;
        cb = cb_hi;
    } else if (p.cut_mode != 0) {
        cb_lo = 0.0; cb_hi = cb = 1.0e15;          // no class given (getters): extents only, no tile logic
    }
    bool compact = !p.uncut && cb < 268435456.0 && (double)c->N + 2.0 * std::ceil(cb) + 8.0 < 2147483647.0;
    p.cb_floor = p.uncut ? 0 : (int64_t)std::fmin(std::floor(cb_lo), 4.0e18);
    p.cb_ceil = p.uncut ? 0 : (int64_t)std::fmin(std::ceil(cb_hi), 4.0e18);
    p.compact = compact ? 1 : 0;
    if (compact) {
        p.kmin = -(p.cb_ceil + 2);
        p.ksent = (int32_t)(c->N + 2 * p.cb_ceil + 6);
    } else {
        p.kmin = -(1LL << 30);
        p.ksent = INT32_MAX;
    }
    p.profile = c->profile;
    p.kappa1 = std::sqrt((double)HK_Z1) * p.beta * 1.001;
    p.kappa2 = std::sqrt((double)HK_Z2) * p.beta * 1.001;
    if (p.profile == HK_PROFILE_LORENTZ) p.kappa1 = p.kappa2 = 0.0;      // no core, no second term: every pair is "far"
    p.inv1p_k1 = 1.0 / (1.0 + p.kappa1); p.inv1m_k1 = 1.0 / (1.0 - p.kappa1);
    p.inv1p_k2 = 1.0 / (1.0 + p.kappa2); p.inv1m_k2 = 1.0 / (1.0 - p.kappa2);
    p.kappaN = p.kappa2; p.inv1p_kN = p.inv1p_k2; p.inv1m_kN = p.inv1m_k2; p.core_nodes = 0;
    p.kappa3 = std::sqrt((double)HK_ZG) * p.beta * 1.005;
    p.inv1p_k3 = 1.0 / (1.0 + p.kappa3); p.inv1m_k3 = 1.0 / (1.0 - p.kappa3);
    p.numin_bins = c->numin / c->dnu;
    p.kb = pick_kb(c, cut);
    p.n_ct = (int32_t)((c->N + 32 * p.kb - 1) / (32 * p.kb));
    p.chunk = chunk;
    p.chunk_node = 16384;
    p.chunk_centre = 2048;
    p.chunk_lane = 16384;
    p.sep = c->node_sep;
    p.plinth = (c->plinth && !p.uncut) ? 1 : 0;
    // Plinth removal subtracts each line's value at its cutting length, evaluated directly: towards the extent ends
    // V - V(cut) is a small fraction of V, and the interpolation error of the node scheme (6e-6 of V at 2 half-widths),
    // which does not cancel against the plinth, would be a large one of the difference.  At 3 half-widths the
    // interpolant is good to ~3e-8 (2.8e-7 at 2.5, 3e-9 at 4: tests/test_nodes.py), below the rounding of the two terms.
    if (p.plinth) p.sep = std::fmax(p.sep, HK_NODE_SEP_PLINTH);
    p.cut_bins = cb;
    p.mode = c->debug_mode;
    return p;
}

// Node hierarchy of this launch: level l has tiles of 32 kb 2^l bins; a level is kept while some line can be both
// separated from one of its tiles (centre >= sep half-widths away) and cover it (centre + cut beyond its far edge).
Levels make_levels(const hk_ctx* c, const Params& p)
{
    Levels lv;
    std::memset(&lv, 0, sizeof(lv));
    lv.w0 = 32 * p.kb;
    if (p.mode != 0 || !(p.sep >= 1.5)) return lv;
    const double reach = p.uncut ? (double)c->N * 2.0 : (double)p.cb_floor;
    int32_t off = 0;
    for (int l = 0; l < kMaxLevels; ++l) {
        const double W = (double)lv.w0 * (double)(1LL << l);
        if (0.5 * W * (p.sep + 1.0) > reach) break;
        const int64_t nt = (c->N + (int64_t)W - 1) / (int64_t)W;
        lv.off[l] = off;
        off += (int32_t)nt;
        lv.n_levels = l + 1;
        if (nt <= 1) break;
    }
    lv.off[lv.n_levels] = off;
    lv.n_entries = off;
    return lv;
}

int32_t pick_chunk(const hk_ctx* c, int64_t n, double cut)
{
    const double tile = 32.0 * pick_kb(c, cut);
    const double n_ct = std::ceil((double)c->N / tile);
    double tiles_per_line = is_uncut(cut) ? n_ct : std::fmin(2.0 * cut / c->dnu / tile + 1.0, n_ct);
    double pairs = (double)n * tiles_per_line;
    double want = pairs / ((double)c->n_sm * 32.0);
    int64_t ch = (int64_t)std::ceil(want / 256.0) * 256;
    if (ch < 512) ch = 512;
    if (ch > 32768) ch = 32768;
    return (int32_t)ch;
}

int bits_for(uint32_t v)
{
    int b = 1;
    while (b < 32 && (v >> b) != 0) ++b;
    return b;
}

__global__ void __launch_bounds__(256) extents_kernel(Params p, const double* __restrict__ nu0, const double* __restrict__ A,
                                                      const double* __restrict__ g, const double* __restrict__ E,
                                                      const double* __restrict__ gam, const double* __restrict__ nx,
                                                      LineExtra ex, int64_t n, int32_t* ilo, int32_t* ihi, int32_t* jc,
                                                      double* S, double* gL, double* aD)
{
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        LineOut o = p.n_iso > 0 ? line_math(p, nu0[i], A[i], g[i], E[i], gam[i], nx[i], ex.gam_self[i], ex.delta[i], ex.iso[i])
                                : line_math(p, nu0[i], A[i], g[i], E[i], gam[i], nx[i]);
        bool live = o.valid && o.ilo <= o.ihi;
        if (ilo) ilo[i] = live ? (int32_t)o.ilo : 0;
        if (ihi) ihi[i] = live ? (int32_t)o.ihi : -1;
        if (jc) jc[i] = o.valid ? (int32_t)max(min(o.jc, (int64_t)INT32_MAX), (int64_t)INT32_MIN) : 0;
        if (S) S[i] = o.S;
        if (gL) gL[i] = o.gammaL;
        if (aD) aD[i] = o.alphaD;
    }
}

// extents and centre bins as the last compute wrote them into its sorted records, back in the caller's line order
__global__ void __launch_bounds__(256) extents_from_records_kernel(const float4* __restrict__ recB, const float4* __restrict__ recN,
                                                                   const int32_t* __restrict__ idx_sorted, int64_t n,
                                                                   int32_t* ilo, int32_t* ihi, int32_t* jc)
{
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const float4 rb = recB[i];
        const int32_t src = idx_sorted[i], lo = __float_as_int(rb.y), hi = __float_as_int(rb.z);
        if (ilo) ilo[src] = hi >= lo ? lo : 0;
        if (ihi) ihi[src] = hi >= lo ? hi : -1;
        if (jc) jc[src] = __float_as_int(recN[i].x);
    }
}

bool lines_ok(const hk_lines* l)
{
    return l && l->nu0 && l->A && l->g_up && l->E_low && l->gamma_ref && l->n_exp;
}

int grid_for(const hk_ctx* c, int64_t n)
{
    int64_t blocks = (n + 255) / 256;
    int64_t cap = (int64_t)c->n_sm * 16;
    return (int)(blocks < 1 ? 1 : (blocks > cap ? cap : blocks));
}

}  // namespace

extern "C" {

int hk_create(double numin, double numax, double dnu, hk_ctx** out)
{
    if (!out) return HK_EINVAL;
    *out = nullptr;
    if (!std::isfinite(numin) || !std::isfinite(numax) || !std::isfinite(dnu)) return HK_EINVAL;
    if (!(dnu > 0.0) || !(numax > numin)) return HK_EINVAL;
    double Nd = std::floor((numax - numin) / dnu + 0.5);
    if (!(Nd >= 1.0) || Nd >= 2147483648.0 - 4096.0) return HK_EINVAL;
    hk_ctx* c = new (std::nothrow) hk_ctx;
    if (!c) return HK_ENOMEM;
    std::memset(c, 0, sizeof(*c));
    c->numin = numin; c->numax = numax; c->dnu = dnu; c->N = (int64_t)Nd;
    c->node_sep = HK_NODE_SEP;
    c->edge_nodes = 1;
    c->single_pass = 1;
    c->core_nodes = 1;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&c->n_sm, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) { delete c; return HK_ECUDA; }
    for (int i = 0; i <= HK_PH_COUNT && e == cudaSuccess; ++i) e = cudaEventCreate(&c->ev[i]);
    for (int i = 0; i < 2 && e == cudaSuccess; ++i) {
        e = cudaEventCreateWithFlags(&c->ev_h2d[i], cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_done[i], cudaEventDisableTiming);
    }
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking);
    if (e != cudaSuccess) { hk_destroy(c); return HK_ECUDA; }
    *out = c;
    return HK_OK;
}

int hk_destroy(hk_ctx* ctx)
{
    if (!ctx) return HK_OK;
    for (int i = 0; i <= HK_PH_COUNT; ++i) if (ctx->ev[i]) cudaEventDestroy(ctx->ev[i]);
    for (int i = 0; i < 2; ++i) {
        if (ctx->ev_h2d[i]) cudaEventDestroy(ctx->ev_h2d[i]);
        if (ctx->ev_done[i]) cudaEventDestroy(ctx->ev_done[i]);
    }
    if (ctx->copy_stream) cudaStreamDestroy(ctx->copy_stream);
    delete ctx;
    return HK_OK;
}

int64_t hk_grid_size(const hk_ctx* ctx) { return ctx ? ctx->N : (int64_t)HK_EINVAL; }

int hk_set_conditions(hk_ctx* ctx, double T_K, double P_atm, double mass_amu, double Q)
{
    if (!ctx) return HK_EINVAL;
    if (!std::isfinite(T_K) || !std::isfinite(P_atm) || !std::isfinite(mass_amu) || !std::isfinite(Q)) return HK_EINVAL;
    if (!(T_K > 0.0) || !(P_atm >= 0.0) || !(mass_amu > 0.0) || !(Q > 0.0)) return HK_EINVAL;
    ctx->T = T_K; ctx->P_atm = P_atm; ctx->mass_amu = mass_amu; ctx->Q = Q;
    ctx->have_cond = true;
    return HK_OK;
}

size_t hk_workspace_bytes(const hk_ctx* ctx, int64_t n_lines)
{
    if (!ctx || n_lines < 0 || n_lines >= 2147483647LL) return 0;
    return make_layout(ctx, n_lines).total;
}

int hk_set_workspace(hk_ctx* ctx, void* dev_ptr, size_t bytes)
{
    if (!ctx || (!dev_ptr && bytes)) return HK_EINVAL;
    if (((uintptr_t)dev_ptr & 255u) != 0) return HK_EINVAL;
    ctx->ws = dev_ptr;
    ctx->ws_bytes = bytes;
    ctx->have_run = false;
    ctx->hint_ready = false;
    return HK_OK;
}

int hk_set_core_nodes(hk_ctx* ctx, int on)
{
    if (!ctx) return HK_EINVAL;
    ctx->core_nodes = on ? 1 : 0;
    return HK_OK;
}

int hk_set_single_pass(hk_ctx* ctx, int on)
{
    if (!ctx) return HK_EINVAL;
    ctx->single_pass = on ? 1 : 0;
    return HK_OK;
}

int hk_set_debug_mode(hk_ctx* ctx, int mode)
{
    if (!ctx || mode < 0 || mode > 3) return HK_EINVAL;
    ctx->debug_mode = mode;
    return HK_OK;
}

int hk_set_node_separation(hk_ctx* ctx, double sep)
{
    // 0 switches the node hierarchy off; closer than the default minus a quarter of a half-width the interpolant leaves the error
    // budget (tests/test_nodes.py)
    if (!ctx || !std::isfinite(sep) || sep < 0.0 || sep > 64.0 || (sep > 0.0 && sep < HK_NODE_SEP - 0.25)) return HK_EINVAL;
    ctx->node_sep = sep;
    return HK_OK;
}

int hk_set_cut_mode(hk_ctx* ctx, int mode)
{
    if (!ctx || mode < HK_CUT_FIXED || mode > HK_CUT_DOPPLER) return HK_EINVAL;
    ctx->cut_mode = mode;
    return HK_OK;
}

int hk_set_profile(hk_ctx* ctx, int profile)
{
    if (!ctx || profile < HK_PROFILE_VOIGT || profile > HK_PROFILE_BINNED_GAUSSIAN) return HK_EINVAL;
    ctx->profile = profile;
    return HK_OK;
}

int hk_set_plinth(hk_ctx* ctx, int on)
{
    if (!ctx) return HK_EINVAL;
    ctx->plinth = on ? 1 : 0;
    return HK_OK;
}

int hk_set_node_kernel(hk_ctx* ctx, int entry_stationary)
{
    if (!ctx) return HK_EINVAL;
    ctx->node_entry_stationary = entry_stationary ? 1 : 0;
    return HK_OK;
}

int hk_set_edge_nodes(hk_ctx* ctx, int on)
{
    if (!ctx) return HK_EINVAL;
    ctx->edge_nodes = on ? 1 : 0;
    return HK_OK;
}

int hk_set_tile_bins(hk_ctx* ctx, int bins_per_lane)
{
    if (!ctx || !(bins_per_lane == 0 || bins_per_lane == 2 || bins_per_lane == 4 || bins_per_lane == 8)) return HK_EINVAL;
    ctx->force_kb = bins_per_lane;
    return HK_OK;
}

static int compute_impl(hk_ctx* ctx, const hk_lines* lines, int64_t n_lines, double cut_cm, double* out_k_dev,
                        cudaStream_t stream, bool zero_out, int reuse = 0, const LineExtra* extra = nullptr,
                        const CutClass* cls = nullptr)
{
    if (!ctx || !out_k_dev || n_lines < 0 || n_lines >= 2147483647LL) return HK_EINVAL;
    if (std::isnan(cut_cm)) return HK_EINVAL;
    if (n_lines > 0 && !lines_ok(lines)) return HK_EINVAL;
    if (!ctx->have_cond || !ctx->ws) return HK_ESTATE;
    const Layout L = make_layout(ctx, n_lines);
    if (ctx->ws_bytes < L.total) return HK_ENOSPC;
    char* ws = (char*)ctx->ws;
    DevStats* st = (DevStats*)(ws + L.stats);
    const int n = (int)n_lines;
    Params p = make_params(ctx, cut_cm, pick_chunk(ctx, n_lines, cls ? cls->bound_hi : cut_cm), extra != nullptr, cls);
    const LineExtra ex = extra ? *extra : LineExtra{nullptr, nullptr, nullptr};
    // (with per-line cutting lengths the tile an extent ends in is not a function of the centre bin alone: the
    //  masked direct edge kernel takes those tiles)
    p.edge_nodes = (L.edge_acc_bytes > 0 && ctx->edge_nodes && p.cut_mode == 0) ? 1 : 0;
    p.lane_tight = ctx->in_batch ? 0 : 1;
    // the core at nodes: plain Voigt profile, fixed cut or none, default kernels, and ranges that serve this condition only
    if (p.profile == HK_PROFILE_VOIGT && p.mode == 0 && p.cut_mode == 0 && !ctx->in_batch && !ctx->node_entry_stationary &&
        ctx->core_nodes) {
        p.core_nodes = 1;
        p.kappaN = std::fmin(std::sqrt((double)HK_ZN) * p.beta * 1.001, p.kappa2);
        p.inv1p_kN = 1.0 / (1.0 + p.kappaN); p.inv1m_kN = 1.0 / (1.0 - p.kappaN);
    }

    // reuse (batched conditions on one resident list): 0 nothing, 1 the order of the lines by centre bin (any change of
    // condition), 2 everything but the Lorentz widths (same T, Q, mass: only the pressure moved)
    const bool reuse_sort = reuse >= 1, widths_only = reuse == 2;
    HK_CUDA(cudaEventRecord(ctx->ev[0], stream));
    if (widths_only) reset_run_kernel<<<1, 1, 0, stream>>>(st);
    else HK_CUDA(cudaMemsetAsync(st, 0, sizeof(DevStats), stream));
    if (zero_out) HK_CUDA(cudaMemsetAsync(out_k_dev, 0, (size_t)ctx->N * sizeof(double), stream));
    ctx->have_run = true;
    ctx->host_totals = false;
    ctx->last_multi = false;
    ctx->last_hitran = extra != nullptr;
    ctx->d_totals = (DevTotals*)(ws + L.totals);
    ctx->last_n = n_lines;
    ctx->last_cut = cut_cm;
    ctx->last_stream = stream;
    ctx->d_stats = st;
    ctx->last_recA = nullptr;
    ctx->regions_done = false;
    ctx->last_sort_bits = 0;
    ctx->last_launches = 0;
    ctx->last_kb = p.kb;
    if (n == 0) {
        for (int i = 1; i <= HK_PH_COUNT; ++i) HK_CUDA(cudaEventRecord(ctx->ev[i], stream));
        return HK_OK;
    }

    int32_t* keys_in = (int32_t*)(ws + L.keys_in);
    int32_t* keys_out = (int32_t*)(ws + L.keys_out);
    int32_t* idx_in = (int32_t*)(ws + L.idx_in);
    int32_t* idx_out = (int32_t*)(ws + L.idx_out);
    RecU* recU = (RecU*)(ws + L.recU);
    float* flo = p.profile == HK_PROFILE_BINNED_GAUSSIAN ? (float*)(ws + L.flo) : nullptr;
    float4* recA = (float4*)(ws + L.recA);
    float4* recB = (float4*)(ws + L.recB);
    float4* recN = (float4*)(ws + L.recN);
    float4* recC = (float4*)(ws + L.recC);
    TileRange* tr = (TileRange*)(ws + L.tr);
    NodeRange* nr = (NodeRange*)(ws + L.nr);
    double* node_acc = (double*)(ws + L.node_acc);
    double* edge_acc = L.edge_acc_bytes ? (double*)(ws + L.edge_acc) : nullptr;
    int32_t* counts = (int32_t*)(ws + L.counts);
    int32_t* prefix = (int32_t*)(ws + L.prefix);
    const Levels lv = make_levels(ctx, p);
    ctx->last_recA = recA; ctx->last_recB = recB; ctx->last_recN = recN; ctx->last_idx = idx_out;
    ctx->last_profile = p.profile;
    ctx->last_levels = lv.n_levels;
    ctx->last_p = p; ctx->last_lv = lv;

    if (widths_only) {
        rewidth_kernel<<<grid_for(ctx, n), 256, 0, stream>>>(p, lines->A, lines->gamma_ref, lines->n_exp, idx_out, st, recA, recB,
                                                            recN, recC);
        HK_CUDA(cudaEventRecord(ctx->ev[HK_PH_PREPROCESS + 1], stream));
        HK_CUDA(cudaEventRecord(ctx->ev[HK_PH_SORT + 1], stream));
        if (lv.n_entries > 0) HK_CUDA(cudaMemsetAsync(node_acc, 0, (size_t)lv.n_entries * kP * sizeof(double), stream));
        HK_CUDA(cudaEventRecord(ctx->ev[HK_PH_RANGES + 1], stream));
        ctx->last_launches = 2;
    } else {
    // a2 (decided first): compact keys (any fixed cut) go through a counting sort with the gather fused into the scatter;
    // the bucket array and the scan's scratch live in the radix sort's scratch, which that path does not use
    const int bits = bits_for((uint32_t)p.ksent);
    size_t cub_bytes = L.cub_bytes;
    const int64_t buckets = (int64_t)p.ksent + 2;
    size_t scan_bytes = 0;
    cub::DeviceScan::ExclusiveSum(nullptr, scan_bytes, (const int32_t*)nullptr, (int32_t*)nullptr, (int)buckets, stream);
    const bool counting = p.compact && buckets < 2147483647LL && align_up((size_t)buckets * 4) + scan_bytes <= L.cub_bytes;
    ctx->last_sort_bits = counting ? 0 : bits;
    int32_t* hist = (counting && !reuse_sort) ? (int32_t*)(ws + L.cub) : nullptr;
    // a1 + a2 in one pass for a list the previous compute on this workspace found sorted (line_sorted_kernel); the two
    // passes below then return at once.  Decided on the device: the launch sequence is the same either way.
    DevHint* hint = (DevHint*)(ws + L.hint);
    if (!ctx->hint_ready) { HK_CUDA(cudaMemsetAsync(hint, 0, sizeof(DevHint), stream)); ctx->hint_ready = true; }
    const bool try_single = ctx->single_pass && hist && !flo && !p.plinth && p.cut_mode == 0 && !cls && p.mode == 0;
    const DevHint* skip = try_single ? hint : nullptr;
    if (try_single) {
        line_sorted_kernel<<<grid_for(ctx, n), 256, 0, stream>>>(p, lines->nu0, lines->A, lines->g_up, lines->E_low,
                                                                lines->gamma_ref, lines->n_exp, ex, n, hint, st, keys_out,
                                                                idx_out, recA, recB, recN, recC);
        single_pass_decide_kernel<<<1, 1, 0, stream>>>(st, hint);
    }
    if (hist) HK_CUDA(cudaMemsetAsync(hist, 0, (size_t)buckets * 4, stream));
    // a1: per-line parameters, keys (and the histogram of the keys)
    line_kernel<<<grid_for(ctx, n), 256, 0, stream>>>(p, lines->nu0, lines->A, lines->g_up, lines->E_low, lines->gamma_ref,
                                                      lines->n_exp, ex, n, recU, keys_in, counting ? nullptr : idx_in, flo, hist, st,
                                                      skip);
    scale_kernel<<<1, 1, 0, stream>>>(st, skip);
    HK_CUDA(cudaEventRecord(ctx->ev[HK_PH_PREPROCESS + 1], stream));
    // the order by centre bin does not depend on (T, P, Q): later conditions of a batch reuse it (hk_compute_batch)
    if (reuse_sort) {
        gather_kernel<<<grid_for(ctx, n), 256, 0, stream>>>(recU, idx_out, flo, n, st, recA, recB, recN, recC, p.profile);
    } else if (counting) {
        void* scan_tmp = ws + L.cub + align_up((size_t)buckets * 4);
        HK_CUDA(cub::DeviceScan::ExclusiveSum(scan_tmp, scan_bytes, (const int32_t*)hist, hist, (int)buckets, stream));
        scatter_kernel<<<grid_for(ctx, n), 256, 0, stream>>>(recU, keys_in, flo, n, hist, st, keys_out, idx_out, recA, recB, recN,
                                                            recC, p.profile, skip);
        // what the next compute may assume (only this path knows whether the list arrived in order)
        hint_update_kernel<<<1, 1, 0, stream>>>(st, hint);
    } else {
        HK_CUDA(cub::DeviceRadixSort::SortPairs(ws + L.cub, cub_bytes, (const int32_t*)keys_in, keys_out,
                                                (const int32_t*)idx_in, idx_out, n, 0, bits, stream));
        gather_kernel<<<grid_for(ctx, n), 256, 0, stream>>>(recU, idx_out, flo, n, st, recA, recB, recN, recC, p.profile);
    }
    HK_CUDA(cudaEventRecord(ctx->ev[HK_PH_SORT + 1], stream));
    // a3: tile ranges, node ranges and work units.  counts = [far | mid | edge | centre | near | node | 0], one scan.
    const int n_counts = 6 * p.n_ct + lv.n_entries + 1;
    int32_t* cnt_far = counts;
    int32_t* cnt_mid = counts + p.n_ct;
    int32_t* cnt_edge = counts + 2 * p.n_ct;
    int32_t* cnt_centre = counts + 3 * p.n_ct;
    int32_t* cnt_near = counts + 4 * p.n_ct;
    int32_t* cnt_lane = counts + 5 * p.n_ct;
    int32_t* cnt_node = counts + 6 * p.n_ct;
    HK_CUDA(cudaMemsetAsync(counts, 0, (size_t)n_counts * 4, stream));
    range_kernel<<<(p.n_ct + 255) / 256, 256, 0, stream>>>(p, lv, keys_out, n, tr, cnt_far, cnt_mid, cnt_edge, cnt_centre,
                                                           cnt_near, cnt_lane, st);
    ctx->last_launches = 4 + (try_single ? 2 : 0) + ((counting && !reuse_sort) ? 1 : 0);   // line, scale, gather / scatter, range (+ single pass and its decision, hint; node range below)
    if (lv.n_entries > 0) {
        HK_CUDA(cudaMemsetAsync(node_acc, 0, (size_t)lv.n_entries * kP * sizeof(double), stream));
        node_range_kernel<<<(lv.n_entries + 255) / 256, 256, 0, stream>>>(p, lv, keys_out, n, tr, nr, cnt_node, st);
        ++ctx->last_launches;
    }
    cub_bytes = L.cub_bytes;
    HK_CUDA(cub::DeviceScan::ExclusiveSum(ws + L.cub, cub_bytes, (const int32_t*)counts, prefix, n_counts, stream));
    HK_CUDA(cudaEventRecord(ctx->ev[HK_PH_RANGES + 1], stream));
    }
    // a4-a7: accumulate
    AccArgs a;
    a.recA = recA; a.recB = recB; a.recN = recN; a.recC = recC; a.tr = tr; a.nr = nr;
    a.prefix_far = prefix; a.prefix_mid = prefix + p.n_ct; a.prefix_edge = prefix + 2 * p.n_ct;
    a.prefix_centre = prefix + 3 * p.n_ct; a.prefix_near = prefix + 4 * p.n_ct;
    a.prefix_lane = prefix + 5 * p.n_ct;
    a.prefix_node = prefix + 6 * p.n_ct;
    a.st = st; a.out_k = out_k_dev; a.node_acc = node_acc; a.profile = p.profile;
    const bool use_edge_nodes = p.edge_nodes && p.mode == 0 && lv.n_levels > 0 && !p.uncut;
    a.edge_acc = use_edge_nodes ? edge_acc : nullptr;
    a.plinth_acc = p.plinth ? (double*)(ws + L.plinth_acc) : nullptr;
    a.N = ctx->N; a.n_ct = p.n_ct; a.chunk = p.chunk; a.chunk_node = p.chunk_node; a.chunk_centre = p.chunk_centre; a.chunk_lane = p.chunk_lane; a.lv = lv;
    const int grid = ctx->n_sm * 2;
    if (lv.n_entries > 0) {
        if (ctx->node_entry_stationary) node_kernel<<<ctx->n_sm * kNodeCtas, kThreads, 0, stream>>>(a);
        else {
            HK_CUDA(cudaFuncSetAttribute(node_lines_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kNLSmemBytes));
            node_lines_kernel<<<ctx->n_sm * kNLCtas, kNLThreads, kNLSmemBytes, stream>>>(p, a);
        }
        ++ctx->last_launches;
    }
    HK_CUDA(cudaEventRecord(ctx->ev[HK_PH_NODE + 1], stream));
    // every CUDA call inside is checked: the first failure is returned and nothing more is enqueued
    auto launch = [&](auto kb_tag) -> cudaError_t {
        constexpr int KB = decltype(kb_tag)::value;
        cudaError_t e = cudaSuccess;
#define HK_TRY(call) do { e = (call); if (e != cudaSuccess) return e; } while (0)
        if (p.mode != 1 && p.mode != 2) { interior_kernel<KB, false><<<grid, kThreads, 0, stream>>>(a); ++ctx->last_launches; }
        HK_TRY(cudaEventRecord(ctx->ev[HK_PH_FAR + 1], stream));
        if (p.mode != 1) { interior_kernel<KB, true><<<grid, kThreads, 0, stream>>>(a); ++ctx->last_launches; }
        HK_TRY(cudaEventRecord(ctx->ev[HK_PH_MID + 1], stream));
        if (p.mode == 0 || p.mode == 3) { edge_kernel<KB><<<ctx->n_sm * 4, kThreads, 0, stream>>>(a); ++ctx->last_launches; }
        if (use_edge_nodes) {
            HK_TRY(cudaMemsetAsync(edge_acc, 0, L.edge_acc_bytes, stream));
            edge_node_kernel<<<ctx->n_sm * 3, kThreads, 0, stream>>>(p, a, keys_out, n);
            const int64_t nsc = 2 * ((ctx->N + lv.w0 - 1) / lv.w0) * kP;
            edge_scan_kernel<<<(int)((nsc + 255) / 256), 256, 0, stream>>>(a);
            edge_bins_kernel<<<(int)((ctx->N + 255) / 256), 256, 0, stream>>>(a);
            ctx->last_launches += 3;
        }
        HK_TRY(cudaGetLastError());
        HK_TRY(cudaEventRecord(ctx->ev[HK_PH_EDGE + 1], stream));
        if (p.mode == 0 || p.mode == 3) {
            // rows (lanes own bins): nothing to do for the Gaussian profiles, whose records carry no Lorentz amplitude
            const bool gauss = p.profile == HK_PROFILE_DOPPLER || p.profile == HK_PROFILE_BINNED_GAUSSIAN;
            if (!gauss) { centre_row_kernel<KB><<<ctx->n_sm * kRowCtas, 32 * kRowWarps, 0, stream>>>(a); ++ctx->last_launches; }
        }
        HK_TRY(cudaEventRecord(ctx->ev[HK_PH_CENTRE + 1], stream));
        if (p.mode == 0 || p.mode == 3) {
            // innermost bins (lane <-> line): none for a pure Lorentzian.  Small CTAs: the pooled visits of a unit are dealt to
            // the CTA's warps in groups of 32 between block-level barriers, and with 8 warps a third of them waited at
            // those barriers (measured on config 4: 8 warps 30.0 ms, 4: 28.4, 2: 27.9, 1: 29.8).  Very sparse lists (fewer
            // than 32 lines per level-0 tile on average) run 1-warp CTAs: a work unit there is a handful of lines
            if (p.profile != HK_PROFILE_LORENTZ) {
                auto lanek = [&](auto binned_tag) {
                    constexpr bool kB = decltype(binned_tag)::value;
                    if ((double)n_lines * (32.0 * KB) < 32.0 * (double)ctx->N)
                        centre_lane_kernel<KB, 1, kB><<<ctx->n_sm * kLaneCtas * 8, 32, 0, stream>>>(a);
                    else
                        centre_lane_kernel<KB, 2, kB><<<ctx->n_sm * kLaneCtas * 4, 64, 0, stream>>>(a);
                };
                if (p.profile == HK_PROFILE_BINNED_GAUSSIAN) lanek(std::true_type());
                else lanek(std::false_type());
                ++ctx->last_launches;
            }
        }
        HK_TRY(cudaEventRecord(ctx->ev[HK_PH_LANE + 1], stream));
        near_kernel<KB><<<grid, kThreads, 0, stream>>>(a);
        ++ctx->last_launches;
        HK_TRY(cudaGetLastError());
        HK_TRY(cudaEventRecord(ctx->ev[HK_PH_NEAR + 1], stream));
#undef HK_TRY
        return e;
    };
    if (p.kb == 8) HK_CUDA(launch(std::integral_constant<int, 8>()));
    else if (p.kb == 4) HK_CUDA(launch(std::integral_constant<int, 4>()));
    else HK_CUDA(launch(std::integral_constant<int, 2>()));
    // downward pass: parents' polynomials onto the children's nodes, level-0 nodes onto the bins
    if (lv.n_entries > 0) {
        for (int l = lv.n_levels - 1; l >= 1; --l) {
            const int nth = (lv.off[l] - lv.off[l - 1]) * kP;
            node_down_kernel<<<(nth + 255) / 256, 256, 0, stream>>>(a, l);
            ++ctx->last_launches;
        }
        node_bins_kernel<<<(int)((ctx->N + 255) / 256), 256, 0, stream>>>(a);
        ++ctx->last_launches;
    }
    // plinth removal: difference array over the sorted lines -> running sum over the bins -> subtract
    if (p.plinth) {
        HK_CUDA(cudaMemsetAsync(a.plinth_acc, 0, (size_t)(ctx->N + 1) * sizeof(double), stream));
        plinth_kernel<<<ctx->n_sm * 8, 256, 0, stream>>>(p, a, recU, (int64_t)n);
        size_t cub_bytes = L.cub_bytes;
        HK_CUDA(cub::DeviceScan::InclusiveSum(ws + L.cub, cub_bytes, (const double*)a.plinth_acc, a.plinth_acc,
                                              (int)(ctx->N + 1), stream));
        plinth_apply_kernel<<<(int)((ctx->N + 255) / 256), 256, 0, stream>>>(a);
        ctx->last_launches += 2;
    }
    HK_CUDA(cudaEventRecord(ctx->ev[HK_PH_DOWN + 1], stream));
    HK_CUDA(cudaGetLastError());
    return HK_OK;
}

// ---- cutting length as a multiple of each line's half-width (L239) ------------------------------------------
// min and max of the per-line cutting length over the lines that have one
__global__ void __launch_bounds__(256) cut_range_kernel(Params p, const double* __restrict__ nu0, const double* __restrict__ A,
                                                        const double* __restrict__ g, const double* __restrict__ E,
                                                        const double* __restrict__ gam, const double* __restrict__ nx,
                                                        LineExtra ex, int64_t n, unsigned long long* __restrict__ mm)
{
    unsigned long long lo = ~0ULL, hi = 0ULL;
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        LineOut o = p.n_iso > 0 ? line_math(p, nu0[i], A[i], g[i], E[i], gam[i], nx[i], ex.gam_self[i], ex.delta[i], ex.iso[i])
                                : line_math(p, nu0[i], A[i], g[i], E[i], gam[i], nx[i]);
        if (!o.valid) continue;
        const double c = p.cut_factor * (p.cut_mode == 1 ? o.gammaL : o.alphaD * 0.83255461115769775635);
        if (!(c > 0.0) || !isfinite(c)) continue;
        const unsigned long long b = (unsigned long long)__double_as_longlong(c);     // positive doubles order as integers
        lo = min(lo, b); hi = max(hi, b);
    }
    for (int o = 16; o > 0; o >>= 1) {
        lo = min(lo, __shfl_xor_sync(0xffffffffu, lo, o));
        hi = max(hi, __shfl_xor_sync(0xffffffffu, hi, o));
    }
    if ((threadIdx.x & 31) == 0) { atomicMin(mm, lo); atomicMax(mm + 1, hi); }
}

// One entry for every compute: fixed cut or uncut -> one pass; width-relative cut -> the range of cutting lengths is
// read back (ONE host synchronisation), then one pass per class [c, 2c) of cutting length, each with its own sort,
// tile ranges and node hierarchy; the passes add into out_k.  A class keeps the ratio of the largest to the
// smallest extent below 2, which is what the interior / node classification of a tile needs to stay useful.
static int compute_any(hk_ctx* ctx, const hk_lines* lines, int64_t n_lines, double cut_cm, double* out_k_dev,
                       cudaStream_t stream, bool zero_out, int reuse = 0, const LineExtra* extra = nullptr)
{
    if (!ctx || ctx->cut_mode == 0 || is_uncut(cut_cm) || n_lines <= 0)
        return compute_impl(ctx, lines, n_lines, cut_cm, out_k_dev, stream, zero_out, reuse, extra);
    if (!out_k_dev || n_lines >= 2147483647LL || std::isnan(cut_cm) || !lines_ok(lines)) return HK_EINVAL;
    if (!ctx->have_cond || !ctx->ws) return HK_ESTATE;
    const Layout L = make_layout(ctx, n_lines);
    if (ctx->ws_bytes < L.total) return HK_ENOSPC;
    unsigned long long* mm = (unsigned long long*)((char*)ctx->ws + L.stats);     // the stats block is free before a pass
    const unsigned long long init[2] = {~0ULL, 0ULL};
    HK_CUDA(cudaMemcpyAsync(mm, init, sizeof(init), cudaMemcpyHostToDevice, stream));
    {
        const Params p = make_params(ctx, cut_cm, 512, extra != nullptr);
        const LineExtra ex = extra ? *extra : LineExtra{nullptr, nullptr, nullptr};
        cut_range_kernel<<<grid_for(ctx, n_lines), 256, 0, stream>>>(p, lines->nu0, lines->A, lines->g_up, lines->E_low,
                                                                     lines->gamma_ref, lines->n_exp, ex, n_lines, mm);
    }
    unsigned long long got[2];
    HK_CUDA(cudaMemcpyAsync(got, mm, sizeof(got), cudaMemcpyDeviceToHost, stream));
    HK_CUDA(cudaStreamSynchronize(stream));
    double cmin, cmax;
    std::memcpy(&cmin, &got[0], 8);
    std::memcpy(&cmax, &got[1], 8);
    const bool none = got[0] == ~0ULL;                     // no line has a positive cutting length
    int64_t launches = 0;
    DevTotals* totals = (DevTotals*)((char*)ctx->ws + L.totals);
    HK_CUDA(cudaMemsetAsync(totals, 0, sizeof(DevTotals), stream));
    int rc = HK_OK;
    bool first = true;
    double lo = none ? 1.0 : cmin;
    const double top = none ? 1.0 : cmax;
    // classes [lo, 2 lo) until the largest cutting length is covered; the 64th class is open-ended (its tile bounds come
    // from [lo, top], correct for any ratio, only less sharp), so no line is ever left out however wide the range
    constexpr int kMaxClasses = 64;
    for (int k = 0; k < kMaxClasses && rc == HK_OK; ++k) {
        CutClass cls;
        cls.first = first;
        cls.lo = first ? 0.0 : lo;
        const bool last = (2.0 * lo > top) || k == kMaxClasses - 1;
        cls.hi = last ? INFINITY : 2.0 * lo;
        cls.bound_lo = lo;
        cls.bound_hi = last ? top : 2.0 * lo;
        rc = compute_impl(ctx, lines, n_lines, cut_cm, out_k_dev, stream, zero_out && first, false, extra, &cls);
        if (rc != HK_OK) break;
        launches += ctx->last_launches;
        add_totals_kernel<<<1, 1, 0, stream>>>(ctx->d_stats, totals);      // per-pass counters summed on the device
        first = false;
        if (!(cls.hi < INFINITY)) break;
        lo *= 2.0;
    }
    if (rc != HK_OK) return rc;
    HK_CUDA(cudaGetLastError());
    ctx->last_launches = launches;
    ctx->host_totals = true;
    ctx->last_multi = true;
    ctx->tot_lines = n_lines;
    return HK_OK;
}

int hk_compute(hk_ctx* ctx, const hk_lines* lines, int64_t n_lines, double cut_cm, double* out_k_dev, void* stream_v)
{
    return compute_any(ctx, lines, n_lines, cut_cm, out_k_dev, (cudaStream_t)stream_v, true);
}

int hk_accumulate(hk_ctx* ctx, const hk_lines* lines, int64_t n_lines, double cut_cm, double* out_k_dev, void* stream_v)
{
    return compute_any(ctx, lines, n_lines, cut_cm, out_k_dev, (cudaStream_t)stream_v, false);
}

}  // extern "C"

// ---- hk_compute_static: the hot path on a workspace nobody allocates -------------------------------------------------
// The workspace of hk_compute is the caller's (hk_set_workspace).  A caller that cannot allocate device memory at all gets
// this one instead: HK_STATIC_WS_BYTES of device memory that belong to the library image (every GPU that loads libhk.so
// holds them until the process exits).  In HOST code the name g_static_ws is a host-side stand-in, not a device address:
// the address the kernels need comes from cudaGetSymbolAddress, once per device, with that device current.
static __device__ __align__(256) unsigned char g_static_ws[HK_STATIC_WS_BYTES];

namespace {
constexpr int kMaxDevices = 64;
void* g_static_ws_addr[kMaxDevices];          // per device ordinal; null until resolved

// -> HK_OK and the device address of g_static_ws on the CURRENT device
int static_ws_address(hk_ctx* ctx, void** out)
{
    int dev = -1;
    HK_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) return HK_EINVAL;
    if (!g_static_ws_addr[dev]) {
        void* p = nullptr;
        HK_CUDA(cudaGetSymbolAddress(&p, g_static_ws));
        if (!p || ((uintptr_t)p & 255u) != 0) return HK_ECUDA;
        g_static_ws_addr[dev] = p;
    }
    *out = g_static_ws_addr[dev];
    return HK_OK;
}
}  // namespace

extern "C" {

int hk_compute_static(hk_ctx* ctx, const hk_lines* lines, int64_t n_lines, double cut_cm, double* out_k_dev, void* stream_v)
{
    if (!ctx || !out_k_dev || n_lines < 0 || n_lines >= 2147483647LL || std::isnan(cut_cm)) return HK_EINVAL;
    if (n_lines > 0 && !lines_ok(lines)) return HK_EINVAL;
    if (!ctx->have_cond) return HK_ESTATE;
    if (ctx->cut_mode != 0 && !is_uncut(cut_cm)) return HK_ESTATE;     // (width-relative cuts read counters back between passes)
    if (make_layout(ctx, n_lines).total > (size_t)HK_STATIC_WS_BYTES) return HK_ENOSPC;
    void* ws = nullptr;
    const int rc_ws = static_ws_address(ctx, &ws);
    if (rc_ws != HK_OK) return rc_ws;
    // the caller's own workspace binding (if any) steps aside for this call.  The static array keeps what the last call on
    // it -- of ANY context -- left there: everything compute_impl needs at zero it clears itself on the stream (counters,
    // work-unit counts, node and extent-end sums, the sort's buckets), and the single-pass hint of the previous call is
    // discarded (hint_ready = false: a list the previous call found sorted is no statement about this one's context)
    void* const ws0 = ctx->ws;
    const size_t bytes0 = ctx->ws_bytes;
    const bool hint0 = ctx->hint_ready;
    ctx->ws = ws; ctx->ws_bytes = (size_t)HK_STATIC_WS_BYTES; ctx->hint_ready = false;
    const int rc = compute_any(ctx, lines, n_lines, cut_cm, out_k_dev, (cudaStream_t)stream_v, true);
    ctx->ws = ws0; ctx->ws_bytes = bytes0; ctx->hint_ready = hint0;
    return rc;
}

int hk_compute_batch(hk_ctx* ctx, const hk_lines* lines, int64_t n_lines, double cut_cm, int32_t n_cond, const double* T_K,
                     const double* P_atm, const double* Q, double* out_k_dev, void* stream_v)
{
    if (!ctx || n_cond < 0 || (n_cond > 0 && (!T_K || !P_atm || !Q || !out_k_dev))) return HK_EINVAL;
    if (!ctx->have_cond || !ctx->ws) return HK_ESTATE;
    for (int32_t c = 0; c < n_cond; ++c) {          // validate everything before enqueueing anything
        if (!std::isfinite(T_K[c]) || !std::isfinite(P_atm[c]) || !std::isfinite(Q[c])) return HK_EINVAL;
        if (!(T_K[c] > 0.0) || !(P_atm[c] >= 0.0) || !(Q[c] > 0.0)) return HK_EINVAL;
    }
    const double T0 = ctx->T, P0 = ctx->P_atm, Q0 = ctx->Q;
    int rc = HK_OK;
    int64_t launches = 0;
    ctx->in_batch = true;
    for (int32_t c = 0; c < n_cond && rc == HK_OK; ++c) {
        ctx->T = T_K[c]; ctx->P_atm = P_atm[c]; ctx->Q = Q[c];
        // what the previous condition of the batch left in the workspace is reused as far as it still holds: the order by
        // centre bin always; everything but the Lorentz widths when only the pressure moved (plain Voigt profile, fixed cut
        // or none, no plinth -- whose kernel reads the unsorted records)
        int reuse = c > 0 ? 1 : 0;
        if (c > 0 && T_K[c] == T_K[c - 1] && Q[c] == Q[c - 1] && ctx->profile == HK_PROFILE_VOIGT && !ctx->plinth &&
            (ctx->cut_mode == 0 || is_uncut(cut_cm)) && ctx->debug_mode == 0)
            reuse = 2;
        rc = compute_any(ctx, lines, n_lines, cut_cm, out_k_dev + (size_t)c * (size_t)ctx->N, (cudaStream_t)stream_v, true,
                         reuse);
        launches += ctx->last_launches;
    }
    ctx->in_batch = false;
    ctx->T = T0; ctx->P_atm = P0; ctx->Q = Q0;
    ctx->last_launches = launches;
    return rc;
}

// ---- host-buffer pipeline ---------------------------------------------------------------
namespace {
constexpr int64_t kDefaultBlock = 1LL << 25;

int64_t host_block(int64_t n_lines, int64_t block_lines)
{
    int64_t b = block_lines > 0 ? block_lines : kDefaultBlock;
    if (b > n_lines) b = n_lines;
    if (b < 1) b = 1;
    if (b > 2147483646LL) b = 2147483646LL;
    return b;
}

struct HostLayout {
    size_t dev_ws, stage[2], k, total;
};

HostLayout make_host_layout(const hk_ctx* c, int64_t n_lines, int64_t block_lines)
{
    const int64_t b = host_block(n_lines, block_lines);
    HostLayout H;
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off += align_up(bytes); return o; };
    H.dev_ws = take(make_layout(c, b).total);
    H.stage[0] = take((size_t)b * 6 * sizeof(double));
    H.stage[1] = take((size_t)b * 6 * sizeof(double));
    H.k = take((size_t)c->N * sizeof(double));
    H.total = off;
    return H;
}
}  // namespace

size_t hk_workspace_bytes_host(const hk_ctx* ctx, int64_t n_lines, int64_t block_lines)
{
    if (!ctx || n_lines < 0) return 0;
    return make_host_layout(ctx, n_lines, block_lines).total;
}

int hk_compute_host(hk_ctx* ctx, const hk_lines* hl, int64_t n_lines, double cut_cm, double* out_k_host,
                    int64_t block_lines, void* stream_v)
{
    if (!ctx || !out_k_host || n_lines < 0 || std::isnan(cut_cm)) return HK_EINVAL;
    if (n_lines > 0 && !lines_ok(hl)) return HK_EINVAL;
    if (ctx->cut_mode != 0 && !is_uncut(cut_cm)) return HK_EINVAL;        // width-relative cuts: device-resident entry points only
    if (!ctx->have_cond || !ctx->ws) return HK_ESTATE;
    const HostLayout H = make_host_layout(ctx, n_lines, block_lines);
    if (ctx->ws_bytes < H.total) return HK_ENOSPC;
    cudaStream_t stream = (cudaStream_t)stream_v;
    const int64_t B = host_block(n_lines, block_lines);
    char* base = (char*)ctx->ws;
    const size_t full_bytes = ctx->ws_bytes;
    double* k_dev = (double*)(base + H.k);
    const double* src[6] = {hl ? hl->nu0 : nullptr, hl ? hl->A : nullptr, hl ? hl->g_up : nullptr,
                            hl ? hl->E_low : nullptr, hl ? hl->gamma_ref : nullptr, hl ? hl->n_exp : nullptr};
    int rc = HK_OK;
    // the per-block device scratch is the front of the caller's workspace
    ctx->ws = base + H.dev_ws;
    ctx->ws_bytes = H.stage[0] - H.dev_ws;
    ctx->hint_ready = false;                     // (the hint lives in the workspace: another base, another hint)
    DevTotals* totals = (DevTotals*)((char*)ctx->ws + make_layout(ctx, 1).totals);   // (fixed offset in every block's layout)
    cudaError_t e = cudaMemsetAsync(k_dev, 0, (size_t)ctx->N * sizeof(double), stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(totals, 0, sizeof(DevTotals), stream);
    const int64_t n_blocks = n_lines > 0 ? (n_lines + B - 1) / B : 0;
    auto enqueue_copy = [&](int64_t b) -> cudaError_t {
        const int s = (int)(b & 1);
        const int64_t l0 = b * B, nb = (l0 + B <= n_lines) ? B : n_lines - l0;
        double* dst = (double*)(base + H.stage[s]);
        cudaError_t ee = cudaSuccess;
        if (b >= 2) ee = cudaStreamWaitEvent(ctx->copy_stream, ctx->ev_done[s], 0);   // staging buffer free again
        for (int f = 0; f < 6 && ee == cudaSuccess; ++f)
            ee = cudaMemcpyAsync(dst + (size_t)f * B, src[f] + l0, (size_t)nb * sizeof(double), cudaMemcpyHostToDevice,
                                 ctx->copy_stream);
        if (ee == cudaSuccess) ee = cudaEventRecord(ctx->ev_h2d[s], ctx->copy_stream);
        return ee;
    };
    if (e == cudaSuccess && n_blocks > 0) e = enqueue_copy(0);
    for (int64_t b = 0; b < n_blocks && e == cudaSuccess && rc == HK_OK; ++b) {
        const int s = (int)(b & 1);
        const int64_t l0 = b * B, nb = (l0 + B <= n_lines) ? B : n_lines - l0;
        if (b + 1 < n_blocks) e = enqueue_copy(b + 1);
        if (e != cudaSuccess) break;
        e = cudaStreamWaitEvent(stream, ctx->ev_h2d[s], 0);
        if (e != cudaSuccess) break;
        double* d = (double*)(base + H.stage[s]);
        hk_lines dl = {d, d + B, d + 2 * B, d + 3 * B, d + 4 * B, d + 5 * B};
        rc = compute_impl(ctx, &dl, nb, cut_cm, k_dev, stream, false);
        if (rc != HK_OK) break;
        e = cudaEventRecord(ctx->ev_done[s], stream);
        if (e != cudaSuccess) break;
        // per-block counters: summed on the device (the stats buffer is reused by the next block), no host synchronisation
        if (ctx->d_stats) add_totals_kernel<<<1, 1, 0, stream>>>(ctx->d_stats, totals);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess && rc == HK_OK)
        e = cudaMemcpyAsync(out_k_host, k_dev, (size_t)ctx->N * sizeof(double), cudaMemcpyDeviceToHost, stream);
    if (e == cudaSuccess && rc == HK_OK) e = cudaStreamSynchronize(stream);
    cudaStreamSynchronize(ctx->copy_stream);
    ctx->ws = base;
    ctx->ws_bytes = full_bytes;
    ctx->hint_ready = false;
    if (rc != HK_OK) return rc;
    if (e != cudaSuccess) return fail_cuda(ctx, e);
    if (n_blocks == 0) { ctx->have_run = true; ctx->last_n = 0; ctx->last_stream = stream; ctx->d_stats = nullptr; }
    ctx->host_totals = true;
    ctx->last_multi = n_blocks > 1;
    ctx->d_totals = totals;
    ctx->tot_lines = n_lines;
    return HK_OK;
}

int hk_get_extents(hk_ctx* ctx, const hk_lines* lines, int64_t n_lines, int32_t* ilo_dev, int32_t* ihi_dev,
                   int32_t* jc_dev, void* stream_v)
{
    if (!ctx || n_lines < 0) return HK_EINVAL;
    if (!ctx->have_cond || !ctx->have_run) return HK_ESTATE;
    cudaStream_t stream = (cudaStream_t)stream_v;
    const bool from_records = ctx->last_recA && !ctx->last_multi && n_lines == ctx->last_n;
    if (from_records) {
        // what the last compute wrote (sorted records, put back in the caller's line order): valid after hk_compute,
        // hk_accumulate, hk_compute_hitran and a single-block hk_compute_host; `lines` is not read
        if (n_lines > 0) {
            if (stream != ctx->last_stream) HK_CUDA(cudaStreamSynchronize(ctx->last_stream));
            extents_from_records_kernel<<<grid_for(ctx, n_lines), 256, 0, stream>>>(ctx->last_recB, ctx->last_recN, ctx->last_idx, n_lines,
                                                                                  ilo_dev, ihi_dev, jc_dev);
            HK_CUDA(cudaGetLastError());
        }
    } else {
        // several passes or blocks shared the record buffer (width-relative cutting lengths, hk_compute_host with more
        // than one block, a different n_lines): recompute from the lines with the conditions and cut of the last compute
        if (ctx->last_hitran) return HK_ESTATE;                  // HITRAN-style lists: hk_get_line_params_hitran
        if (n_lines > 0 && !lines_ok(lines)) return HK_EINVAL;
        if (n_lines > 0) {
            const Params p = make_params(ctx, ctx->last_cut, 512);
            extents_kernel<<<grid_for(ctx, n_lines), 256, 0, stream>>>(p, lines->nu0, lines->A, lines->g_up, lines->E_low,
                                                                       lines->gamma_ref, lines->n_exp, LineExtra{nullptr, nullptr, nullptr},
                                                                       n_lines, ilo_dev, ihi_dev, jc_dev, nullptr, nullptr, nullptr);
            HK_CUDA(cudaGetLastError());
        }
    }
    HK_CUDA(cudaStreamSynchronize(stream));
    return HK_OK;
}

int hk_get_line_params(hk_ctx* ctx, const hk_lines* lines, int64_t n_lines, double* S_dev, double* gammaL_dev,
                       double* alphaD_dev, void* stream_v)
{
    if (!ctx || n_lines < 0 || (n_lines > 0 && !lines_ok(lines))) return HK_EINVAL;
    if (!ctx->have_cond) return HK_ESTATE;
    cudaStream_t stream = (cudaStream_t)stream_v;
    if (n_lines > 0) {
        const Params p = make_params(ctx, 0.0, 512);
        extents_kernel<<<grid_for(ctx, n_lines), 256, 0, stream>>>(p, lines->nu0, lines->A, lines->g_up, lines->E_low,
                                                                   lines->gamma_ref, lines->n_exp, LineExtra{nullptr, nullptr, nullptr},
                                                                   n_lines, nullptr, nullptr, nullptr, S_dev, gammaL_dev, alphaD_dev);
        HK_CUDA(cudaGetLastError());
    }
    HK_CUDA(cudaStreamSynchronize(stream));
    return HK_OK;
}

// ---- bands of different resolution (L218) ---------------------------------------------------
int hk_compute_bands(hk_ctx* const* ctxs, int32_t n_bands, const hk_lines* lines, int64_t n_lines, double cut_cm,
                     double* const* out_k_dev, void* stream_v)
{
    if (n_bands < 0 || (n_bands > 0 && (!ctxs || !out_k_dev))) return HK_EINVAL;
    for (int32_t b = 0; b < n_bands; ++b) {
        if (!ctxs[b] || !out_k_dev[b]) return HK_EINVAL;
        if (!ctxs[b]->have_cond || !ctxs[b]->ws) return HK_ESTATE;
    }
    for (int32_t b = 0; b < n_bands; ++b) {
        const int rc = compute_any(ctxs[b], lines, n_lines, cut_cm, out_k_dev[b], (cudaStream_t)stream_v, true);
        if (rc != HK_OK) return rc;
    }
    return HK_OK;
}

// ---- HITRAN-style inputs ------------------------------------------------------------------
namespace {
bool hitran_ok(const hk_lines_hitran* l)
{
    return l && l->nu0 && l->A && l->g_up && l->E_low && l->gamma_air && l->gamma_self && l->n_exp && l->delta && l->iso;
}
hk_lines as_lines(const hk_lines_hitran* l)
{
    return hk_lines{l->nu0, l->A, l->g_up, l->E_low, l->gamma_air, l->n_exp};
}
}  // namespace

int hk_set_conditions_hitran(hk_ctx* ctx, double T_K, double P_atm, double P_self_atm, int32_t n_iso, const double* mass_amu,
                             const double* Q, const double* abundance)
{
    if (!ctx || n_iso < 1 || n_iso > kMaxIso || !mass_amu || !Q || !abundance) return HK_EINVAL;
    if (!std::isfinite(T_K) || !std::isfinite(P_atm) || !std::isfinite(P_self_atm)) return HK_EINVAL;
    if (!(T_K > 0.0) || !(P_atm >= 0.0) || !(P_self_atm >= 0.0) || !(P_self_atm <= P_atm)) return HK_EINVAL;
    for (int j = 0; j < n_iso; ++j) {
        if (!std::isfinite(mass_amu[j]) || !std::isfinite(Q[j]) || !std::isfinite(abundance[j])) return HK_EINVAL;
        if (!(mass_amu[j] > 0.0) || !(Q[j] > 0.0) || !(abundance[j] >= 0.0)) return HK_EINVAL;
    }
    ctx->T = T_K; ctx->P_atm = P_atm; ctx->P_self = P_self_atm; ctx->n_iso = n_iso;
    for (int j = 0; j < n_iso; ++j) { ctx->iso_mass[j] = mass_amu[j]; ctx->iso_Q[j] = Q[j]; ctx->iso_ab[j] = abundance[j]; }
    ctx->mass_amu = mass_amu[0]; ctx->Q = Q[0];           // the ExoMol-style entry points see isotopologue 0
    ctx->have_cond = true;
    ctx->have_hitran = true;
    return HK_OK;
}

int hk_compute_hitran(hk_ctx* ctx, const hk_lines_hitran* lines, int64_t n_lines, double cut_cm, double* out_k_dev,
                      void* stream_v)
{
    if (!ctx || n_lines < 0 || (n_lines > 0 && !hitran_ok(lines))) return HK_EINVAL;
    if (!ctx->have_hitran) return HK_ESTATE;
    hk_lines base = n_lines > 0 ? as_lines(lines) : hk_lines{nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    LineExtra ex = n_lines > 0 ? LineExtra{lines->gamma_self, lines->delta, lines->iso} : LineExtra{nullptr, nullptr, nullptr};
    return compute_any(ctx, &base, n_lines, cut_cm, out_k_dev, (cudaStream_t)stream_v, true, false, &ex);
}

int hk_get_line_params_hitran(hk_ctx* ctx, const hk_lines_hitran* lines, int64_t n_lines, double cut_cm, double* S_dev,
                              double* gammaL_dev, double* alphaD_dev, int32_t* ilo_dev, int32_t* ihi_dev, int32_t* jc_dev,
                              void* stream_v)
{
    if (!ctx || n_lines < 0 || (n_lines > 0 && !hitran_ok(lines)) || std::isnan(cut_cm)) return HK_EINVAL;
    if (!ctx->have_hitran) return HK_ESTATE;
    cudaStream_t stream = (cudaStream_t)stream_v;
    if (n_lines > 0) {
        const Params p = make_params(ctx, cut_cm, 512, true);
        extents_kernel<<<grid_for(ctx, n_lines), 256, 0, stream>>>(p, lines->nu0, lines->A, lines->g_up, lines->E_low,
                                                                   lines->gamma_air, lines->n_exp,
                                                                   LineExtra{lines->gamma_self, lines->delta, lines->iso},
                                                                   n_lines, ilo_dev, ihi_dev, jc_dev, S_dev, gammaL_dev,
                                                                   alphaD_dev);
        HK_CUDA(cudaGetLastError());
    }
    HK_CUDA(cudaStreamSynchronize(stream));
    return HK_OK;
}

int hk_get_stats(hk_ctx* ctx, hk_stats* host_out)
{
    if (!ctx || !host_out) return HK_EINVAL;
    if (!ctx->have_run) return HK_ESTATE;
    DevStats d;
    std::memset(&d, 0, sizeof(d));
    HK_CUDA(cudaStreamSynchronize(ctx->last_stream));
    if (ctx->d_stats && ctx->last_recA && !ctx->regions_done && ctx->last_n > 0) {
        // per-region evaluation counts, derived from the records on demand (kept out of the hot path)
        const int64_t nl = ctx->last_n;                 // (block pipelines and class passes: the last block / pass)
        if (nl > 0) {
            region_stats_kernel<<<grid_for(ctx, nl), 256, 0, ctx->last_stream>>>(ctx->last_recA, ctx->last_recB, nl, ctx->last_profile,
                                                                                 ctx->last_kb, ctx->d_stats);
            if (ctx->last_p.core_nodes && ctx->last_lv.n_levels > 0)
                core_nodes_stats_kernel<<<grid_for(ctx, nl), 256, 0, ctx->last_stream>>>(ctx->last_p, ctx->last_lv, ctx->last_recA,
                                                                                      ctx->last_recB, ctx->last_recN, nl, ctx->d_stats);
            HK_CUDA(cudaStreamSynchronize(ctx->last_stream));
        }
        ctx->regions_done = true;
    }
    if (ctx->d_stats) HK_CUDA(cudaMemcpy(&d, ctx->d_stats, sizeof(d), cudaMemcpyDeviceToHost));
    std::memset(host_out, 0, sizeof(*host_out));
    host_out->n_lines = ctx->last_n;
    host_out->n_skipped = (int64_t)d.n_skipped;
    host_out->n_off_grid = (int64_t)d.n_off_grid;
    host_out->n_evals = (int64_t)d.n_evals;
    host_out->n_evals_far = (int64_t)(d.n_evals - d.n_cnt_mid);
    host_out->n_evals_mid = (int64_t)(d.n_cnt_mid - d.n_cnt_core);
    host_out->n_evals_core = (int64_t)d.n_cnt_core;
    host_out->n_evals_gh6 = (int64_t)(d.n_cnt_gh6 - d.n_cnt_trap);
    host_out->n_evals_trap = (int64_t)d.n_cnt_trap;
    host_out->n_evals_gh10 = (int64_t)d.n_cnt_gh10;
    host_out->n_units_far = (int64_t)d.units_far;
    host_out->n_units_mid = (int64_t)d.units_mid;
    host_out->n_units_near = (int64_t)d.units_near;
    host_out->n_pairs_mid = (int64_t)d.pairs_mid;
    host_out->bins_per_lane = ctx->last_kb;
    host_out->n_pairs_far = (int64_t)d.pairs_far;
    host_out->n_pairs_near = (int64_t)d.pairs_near;
    host_out->n_launches = ctx->last_launches;
    host_out->n_units_node = (int64_t)d.units_node;
    host_out->n_units_edge = (int64_t)d.units_edge;
    host_out->n_units_centre = (int64_t)d.units_centre;
    host_out->n_pairs_edge = (int64_t)d.pairs_edge;
    host_out->n_pairs_centre = (int64_t)d.pairs_centre;
    host_out->n_pairs_node = (int64_t)d.pairs_node;
    host_out->n_pairs_edge_node = (int64_t)d.pairs_edge_node;
    host_out->n_bins_node = (int64_t)d.bins_node;
    host_out->n_levels = ctx->last_levels;
    host_out->scale_exp = d.scale_exp;
    host_out->sort_bits = ctx->last_sort_bits;
    host_out->n_plinth_illcond = (int64_t)d.n_plinth_illcond;
    host_out->n_unsorted = (int64_t)d.n_unsorted;
    host_out->single_pass = d.single_pass;
    host_out->n_pairs_node_far = (int64_t)d.pairs_node_far;
    host_out->n_pairs_node_core = (int64_t)d.pairs_node_core;
    host_out->n_pairs_node_eval = (int64_t)d.pairs_node_eval;
    host_out->n_evals_gh10_row = (int64_t)d.n_cnt_gh10_row;
    host_out->n_evals_core_nodes = (int64_t)d.n_cnt_core_nodes;
    if (ctx->host_totals) {
        DevTotals t;
        std::memset(&t, 0, sizeof(t));
        if (ctx->d_totals && ctx->tot_lines > 0) HK_CUDA(cudaMemcpy(&t, ctx->d_totals, sizeof(t), cudaMemcpyDeviceToHost));
        host_out->n_lines = ctx->tot_lines;
        host_out->n_skipped = (int64_t)t.n_skipped;
        host_out->n_off_grid = (int64_t)t.n_off_grid;
        host_out->n_evals = (int64_t)t.n_evals;
        host_out->n_plinth_illcond = (int64_t)t.n_plinth_illcond;
    }
    return HK_OK;
}

int hk_get_phase_ms(hk_ctx* ctx, float* out_ms)
{
    if (!ctx || !out_ms) return HK_EINVAL;
    if (!ctx->have_run) return HK_ESTATE;
    HK_CUDA(cudaStreamSynchronize(ctx->last_stream));
    for (int i = 0; i < HK_PH_COUNT; ++i) {
        out_ms[i] = 0.f;
        if (ctx->last_n > 0 || !ctx->host_totals) HK_CUDA(cudaEventElapsedTime(&out_ms[i], ctx->ev[i], ctx->ev[i + 1]));
    }
    return HK_OK;
}

int hk_probe_fp32_ops(int kind, int iters, double* lane_ops_per_s, double* sm_clock_mhz, float* ms_out, void* stream_v)
{
    if (iters < 1 || kind < 0 || kind > 5 || !lane_ops_per_s) return HK_EINVAL;
    cudaStream_t stream = (cudaStream_t)stream_v;
    int dev = 0, n_sm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return HK_ECUDA;
    if (cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return HK_ECUDA;
    float* sink = nullptr;
    long long* clk = nullptr;
    if (cudaMalloc(&sink, sizeof(float)) != cudaSuccess) return HK_ECUDA;
    if (cudaMalloc(&clk, 2 * sizeof(long long)) != cudaSuccess) { cudaFree(sink); return HK_ECUDA; }
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int blocks = n_sm * 4, threads = 512;
    for (int rep = 0; rep < 2; ++rep) {      // first launch warms up
        cudaEventRecord(e0, stream);
        switch (kind) {
            case 0: fp32_probe_kernel<0><<<blocks, threads, 0, stream>>>(iters, sink, clk); break;
            case 1: fp32_probe_kernel<1><<<blocks, threads, 0, stream>>>(iters, sink, clk); break;
            case 2: fp32_probe_kernel<2><<<blocks, threads, 0, stream>>>(iters, sink, clk); break;
            case 3: fp32_probe_kernel<3><<<blocks, threads, 0, stream>>>(iters, sink, clk); break;
            case 4: fp32_probe_kernel<4><<<blocks, threads, 0, stream>>>(iters, sink, clk); break;
            default: fp32_probe_kernel<5><<<blocks, threads, 0, stream>>>(iters, sink, clk); break;
        }
        cudaEventRecord(e1, stream);
    }
    cudaError_t e = cudaStreamSynchronize(stream);
    float ms = 0.f;
    long long h[2] = {0, 1};
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    if (e == cudaSuccess) e = cudaMemcpy(h, clk, sizeof(h), cudaMemcpyDeviceToHost);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(sink); cudaFree(clk);
    if (e != cudaSuccess) return HK_ECUDA;
    // 16 chains x 2 floats per step (MUFU: 16 x 1)
    const double ops = (double)blocks * threads * (double)iters * (kind == 5 ? 16.0 : 32.0);
    *lane_ops_per_s = ops / ((double)ms * 1e-3);
    if (sm_clock_mhz) *sm_clock_mhz = h[1] > 0 ? (double)h[0] / (double)h[1] * 1e3 : 0.0;
    if (ms_out) *ms_out = ms;
    return HK_OK;
}

int hk_probe_fp32_peak(int packed, int iters, double* flops_out, float* ms_out, void* stream_v)
{
    if (!flops_out) return HK_EINVAL;
    double ops = 0.0;
    const int rc = hk_probe_fp32_ops(packed ? 0 : 1, iters, &ops, nullptr, ms_out, stream_v);
    *flops_out = 2.0 * ops;                   // 2 FLOP per FMA
    return rc;
}

int hk_eval_voigt_f32(const float* x_dev, const float* y_dev, int64_t n, float* out_dev, int32_t* region_out_dev,
                      void* stream_v)
{
    if (n < 0 || (n > 0 && (!x_dev || !y_dev || !out_dev))) return HK_EINVAL;
    if (n == 0) return HK_OK;
    int64_t blocks = (n + 255) / 256;
    if (blocks > 65535) blocks = 65535;
    probe_kernel<<<(int)blocks, 256, 0, (cudaStream_t)stream_v>>>(x_dev, y_dev, n, out_dev, region_out_dev);
    return cudaGetLastError() == cudaSuccess ? HK_OK : HK_ECUDA;
}

int hk_last_cuda_error(const hk_ctx* ctx) { return ctx ? ctx->cuda_err : 0; }

const char* hk_strerror(int status)
{
    switch (status) {
        case HK_OK: return "ok";
        case HK_EINVAL: return "invalid argument";
        case HK_ESTATE: return "call out of order (conditions / workspace / compute missing)";
        case HK_ENOSPC: return "workspace too small (hk_compute_static: problem larger than HK_STATIC_WS_BYTES)";
        case HK_ECUDA: return "CUDA call failed (see hk_last_cuda_error)";
        case HK_ENOMEM: return "host allocation failed";
        default: return "unknown status";
    }
}

}  // extern "C"
