// hk_accumulate.cuh -- steps a4-a7 of the hot path: the accumulation kernels.
//
// All are output-stationary: a CTA owns a tile of 32*KB consecutive bins, every warp of the CTA
// holds the SAME bins (a lane owns bins lane + 32 j, j < KB, in registers) and the warps split the
// LINES of each staged batch between them; their partial sums are combined through shared memory
// at the end of a work unit and reach k(nu) with one fp64 atomic per bin per unit.
// Lines arrive sorted by centre bin, so the lines that can reach a tile are one contiguous index
// range, split by range_kernel into
//   [A0,FL0) left-edge | [FL0,NL) node-handled | [NL,FL1) far | [FL1,ML1) mid | [ML1,MR0) centre |
//   [MR0,FR0) mid | [FR0,NR) far | [NR,FR1) node-handled | [FR1,A1) right-edge     (TileRange, hk_device.cuh)
// Node-handled pairs (tile separated from the line) are evaluated at Chebyshev nodes
// by node_kernel on a binary hierarchy of tiles and interpolated onto the bins at the end.
// A work unit is (tile, chunk of a kernel's own classes); units are handed out by an atomic counter to a
// persistent grid (a multiple of the SM count).  fp32 partial sums are flushed into fp64 registers
// every kFlush lines.
//
//   node_kernel               (a5)        : separated (line, tile) pairs at the tile's 8 Chebyshev nodes, every level of
//        the hierarchy; node_down_kernel / node_bins_kernel bring the node sums down to the bins.
//   interior_kernel<KB,false> (a5, "far") : pairs whose whole tile is inside the extent and has
//        |z|^2 >= Z1: branch-free Lorentzian, two lines share one reciprocal, packed fp32 (FFMA2).
//   interior_kernel<KB,true>  (a5, "mid") : same shape, |z|^2 >= Z2: two-term asymptotic, mask-free.
//   edge_node_kernel          (a4)        : extent ends in separated tiles, at the tile's nodes into per-bin accumulators
//        (edge_scan_kernel, edge_bins_kernel finish); edge_kernel<KB>: the masked direct form for the other ends.
//   centre_kernel<KB,W,binned> (a4)       : tiles inside the extent that hold a line's core.  Row pass (Gauss-Hermite 4
//        or two-term rows) + lane pass for |z| < 8 on batches counting-sorted by y.  The dominant kernel.
//   near_kernel<KB>           (a4)        : the generic remainder (tiles partly outside the extent that hold core
//        bins).  Row pass: exact integer extent mask + two-term asymptotic where |z|^2 >= Z2, and the core
//        evaluator in place for lines whose core spans >= 16 bins.  Lane pass, for narrower cores: lanes
//        walk lines, each lane evaluates its own line's core bins; equal bins are combined in the
//        warp and added to a bin tile staged in shared memory.
//   plinth_kernel             (optional)  : the per-line plinths as a difference array, summed over the bins by CUB.
//
// The paper's kernel (L243-330) walks lines in threads and nu-points serially with a
// shared-memory K_s and four launches per block (AL/AR/B/C, L354); what is kept is the idea
// of formula-uniform launches and of partial arrays merged at the end (L254-258, L268).
#pragma once
#include "hk_preprocess.cuh"

namespace hk {

struct AccArgs {
    const float4* __restrict__ recA;
    const float4* __restrict__ recB;
    const float4* __restrict__ recN;
    const float4* __restrict__ recC;           // { dnu/alpha_D, -f dnu/alpha_D, y^2, 1/(cK y) }: the centre kernels' per-line part
    const TileRange* __restrict__ tr;
    const NodeRange* __restrict__ nr;
    // exclusive scans of the work-unit counts (one concatenated scan; each kernel reads its own slice, whose first
    // element is the slice's base): n_ct + 1 entries for the direct kernels, n_entries + 1 for the node kernel
    const int32_t* __restrict__ prefix_far;
    const int32_t* __restrict__ prefix_mid;
    const int32_t* __restrict__ prefix_edge;
    const int32_t* __restrict__ prefix_centre;
    const int32_t* __restrict__ prefix_lane;   // the same line ranges in longer chunks (centre_lane_kernel)
    const int32_t* __restrict__ prefix_near;
    const int32_t* __restrict__ prefix_node;
    DevStats* st;
    double* __restrict__ out_k;
    double* __restrict__ node_acc;             // n_entries x kP node sums (scaled), fp64
    double* __restrict__ plinth_acc;           // N + 1 doubles: difference array of the plinths, then its running sum; or null
    double* __restrict__ edge_acc;             // [2][N][kP] per-bin node sums of extent ends (scaled), fp64; or null
    int64_t N;
    int32_t n_ct, chunk, chunk_node, chunk_centre, chunk_lane;
    int32_t profile;                           // HK_PROFILE_*: only the binned Gaussian changes the kernels' core evaluation
    Levels lv;
};

// Which tile does unit u belong to?  Largest ct with prefix[ct] <= u (u already includes the slice base prefix[0]).
__device__ __forceinline__ int find_tile(const int32_t* __restrict__ prefix, int n_ct, int u)
{
    int lo = 0, hi = n_ct;   // invariant: prefix[lo] <= u < prefix[hi]
    while (hi - lo > 1) {
        int mid = (lo + hi) >> 1;
        if (prefix[mid] <= u) lo = mid; else hi = mid;
    }
    return lo;
}

__device__ __forceinline__ int next_unit(unsigned int* counter, int* s_unit)
{
    __syncthreads();
    if (threadIdx.x == 0) *s_unit = (int)atomicAdd(counter, 1u);
    __syncthreads();
    return *s_unit;
}

__device__ __forceinline__ float2 bcast2(float v) { return make_float2(v, v); }
__device__ __forceinline__ float2 rcp2(float2 q) { return make_float2(rcp_approx(q.x), rcp_approx(q.y)); }

// this warp's share [w0, w1) of the lines [0, n): contiguous, even-sized (pairs stay together)
__device__ __forceinline__ void warp_share(int n, int warp, int& w0, int& w1)
{
    const int per = ((n + 2 * kWarps - 1) / (2 * kWarps)) * 2;
    w0 = min(warp * per, n);
    w1 = min(w0 + per, n);
}

// combine the warps' partial sums (red aliases the staging buffers: call after a __syncthreads that
// follows the last read of them) and add the tile to k(nu)
template <int KB, int W = kWarps>
__device__ __forceinline__ void flush_tile(double* red, const double (&v)[KB], int64_t ct0, const AccArgs& a)
{
    constexpr int kWarps = W;
    constexpr int kTB = 32 * KB;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int j = 0; j < KB; ++j) red[warp * kTB + lane + 32 * j] = v[j];
    __syncthreads();
    for (int i = threadIdx.x; i < kTB; i += 32 * kWarps) {
        double s = 0.0;
#pragma unroll
        for (int w = 0; w < kWarps; ++w) s += red[w * kTB + i];
        const int64_t b = ct0 + i;
        s *= scalbn(1.0, -a.st->scale_exp);
        if (b < a.N && s != 0.0) atomicAdd(a.out_k + b, s);
    }
}

// ---------------------------------------------------------------------------------------
// interior kernels (far: kMid = false, mid: kMid = true)
// ---------------------------------------------------------------------------------------
constexpr int kSubI = 1024;            // lines per staged batch (double-buffered)
constexpr int kLPT = kSubI / kThreads; // lines each thread stages per batch

template <int KB, bool kMid>
__global__ void __launch_bounds__(kThreads, 2) interior_kernel(AccArgs a)
{
    constexpr int kTB = 32 * KB;          // bins per tile
    constexpr int M = KB / 2;             // float2 accumulators per lane
    static_assert(sizeof(double) * kWarps * kTB <= sizeof(float4) * 2 * kSubI, "red must fit in the staging buffers");
    __shared__ float4 sm[2][kSubI];       // { -tl, G2, c, 1.5 a2 }, tl = centre position relative to the tile
    __shared__ int s_unit;
    double* red = reinterpret_cast<double*>(&sm[0][0]);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int32_t* __restrict__ prefix = kMid ? a.prefix_mid : a.prefix_far;
    const int base = prefix[0], total = prefix[a.n_ct];
    unsigned int* counter = kMid ? &a.st->unit_counter_mid : &a.st->unit_counter_far;

    float2 tb[M];
#pragma unroll
    for (int m = 0; m < M; ++m) {
        float b0 = (float)(lane + 64 * m);
        tb[m] = make_float2(b0, b0 + 32.0f);
    }

    for (;;) {
        const int u = next_unit(counter, &s_unit) + base;
        if (u >= total) break;
        const int ct = find_tile(prefix, a.n_ct, u);
        const int64_t ct0 = (int64_t)ct * kTB;
        const TileRange r = a.tr[ct];
        // left and right segments of this class walked as one list; this unit takes lines [v_lo, v_hi) of it
        const int sl0 = kMid ? r.FL1 : r.NL, sl1 = kMid ? r.ML1 : r.FL1;
        const int sr0 = kMid ? r.MR0 : r.FR0, sr1 = kMid ? r.FR0 : r.NR;
        const int v_lo = (u - prefix[ct]) * a.chunk;
        const int v_hi = min(v_lo + a.chunk, (sl1 - sl0) + (sr1 - sr0));
        const int l0 = min(sl0 + v_lo, sl1), l1 = min(sl0 + v_hi, sl1);
        const int r0 = sr0 + max(v_lo - (sl1 - sl0), 0), r1 = sr0 + max(v_hi - (sl1 - sl0), 0);
        const int nl = l1 - l0, nt = nl + (r1 - r0);
        if (nt <= 0) continue;
        if (threadIdx.x == 0) atomicAdd(kMid ? &a.st->units_mid : &a.st->units_far, 1ULL);

        float2 acc[M];
        double acc64[KB];
#pragma unroll
        for (int m = 0; m < M; ++m) acc[m] = make_float2(0.f, 0.f);
#pragma unroll
        for (int j = 0; j < KB; ++j) acc64[j] = 0.0;
        int since_flush = 0;

        float4 pre[kLPT];
        float prea[kLPT];
        auto fetch = [&](int v0) {            // global loads of batch [v0, v0 + kSubI) into registers
#pragma unroll
            for (int k = 0; k < kLPT; ++k) {
                const int v = v0 + threadIdx.x + k * kThreads;
                if (v < nt) {
                    const int li = v < nl ? l0 + v : r0 + (v - nl);
                    pre[k] = a.recA[li];
                    if (kMid) prea[k] = a.recB[li].x;
                }
            }
        };
        auto stash = [&](int v0, int buf) {   // convert to tile-relative records in shared memory
#pragma unroll
            for (int k = 0; k < kLPT; ++k) {
                const int i = threadIdx.x + k * kThreads;
                if (v0 + i < nt) {
                    const float tl = (float)((int64_t)__float_as_int(pre[k].x) - ct0) + pre[k].y;
                    sm[buf][i] = make_float4(-tl, pre[k].z, pre[k].w, kMid ? 1.5f * prea[k] : 0.f);
                }
            }
        };
        fetch(0);
        stash(0, 0);
        __syncthreads();
        int buf = 0;
        for (int v0 = 0; v0 < nt; v0 += kSubI, buf ^= 1) {
            const bool more = v0 + kSubI < nt;
            if (more) fetch(v0 + kSubI);
            const float4* __restrict__ smb = sm[buf];
            int l, le;
            warp_share(min(kSubI, nt - v0), warp, l, le);
            while (l < le) {
                const int stop = min(le, l + (kFlush - since_flush));
                since_flush += stop - l;
                if (!kMid) {
                    for (; l + 1 < stop; l += 2) {
                        const float4 r1 = smb[l], r2 = smb[l + 1];
                        const float2 n1 = bcast2(r1.x), g1 = bcast2(r1.y), c1 = bcast2(r1.z);
                        const float2 n2 = bcast2(r2.x), g2 = bcast2(r2.y), c2 = bcast2(r2.z);
#pragma unroll
                        for (int m = 0; m < M; ++m) {
                            // c1/q1 + c2/q2 = (c1 q2 + c2 q1) / (q1 q2): one reciprocal for two lines
                            const float2 t1 = __fadd2_rn(tb[m], n1);
                            const float2 t2 = __fadd2_rn(tb[m], n2);
                            const float2 q1 = __ffma2_rn(t1, t1, g1);
                            const float2 q2 = __ffma2_rn(t2, t2, g2);
                            const float2 pp = __fmul2_rn(q1, q2);
                            float2 nn = __fmul2_rn(c1, q2);
                            nn = __ffma2_rn(c2, q1, nn);
                            acc[m] = __ffma2_rn(nn, rcp2(pp), acc[m]);
                        }
                    }
                    if (l < stop) {       // odd line out
                        const float4 r1 = smb[l];
                        const float2 n1 = bcast2(r1.x), g1 = bcast2(r1.y), c1 = bcast2(r1.z);
#pragma unroll
                        for (int m = 0; m < M; ++m) {
                            const float2 t1 = __fadd2_rn(tb[m], n1);
                            const float2 q1 = __ffma2_rn(t1, t1, g1);
                            acc[m] = __ffma2_rn(c1, rcp2(q1), acc[m]);
                        }
                        ++l;
                    }
                } else {
                    for (; l < stop; ++l) {
                        // c r (1 + r (A1 - A2 r)),  A1 = 1.5 a^2, A2 = 2 a^2 G^2 = (4/3) A1 G^2
                        const float4 r1 = smb[l];
                        const float2 n1 = bcast2(r1.x), g1 = bcast2(r1.y), c1 = bcast2(r1.z);
                        const float2 A1 = bcast2(r1.w), one = bcast2(1.0f);
                        const float2 nA2 = bcast2(-1.33333333f * r1.w * r1.y);
#pragma unroll
                        for (int m = 0; m < M; ++m) {
                            const float2 t1 = __fadd2_rn(tb[m], n1);
                            const float2 q1 = __ffma2_rn(t1, t1, g1);
                            const float2 rr = rcp2(q1);
                            const float2 uu = __ffma2_rn(nA2, rr, A1);
                            const float2 vv = __ffma2_rn(uu, rr, one);
                            const float2 ww = __fmul2_rn(rr, vv);
                            acc[m] = __ffma2_rn(c1, ww, acc[m]);
                        }
                    }
                }
                if (since_flush >= kFlush) {
#pragma unroll
                    for (int m = 0; m < M; ++m) {
                        acc64[2 * m] += (double)acc[m].x;
                        acc64[2 * m + 1] += (double)acc[m].y;
                        acc[m] = make_float2(0.f, 0.f);
                    }
                    since_flush = 0;
                }
            }
            if (more) stash(v0 + kSubI, buf ^ 1);
            __syncthreads();
        }
        double v[KB];
#pragma unroll
        for (int m = 0; m < M; ++m) {            // acc[m] holds bins lane + 64 m and lane + 64 m + 32: rows 2m and 2m+1
            v[2 * m] = acc64[2 * m] + (double)acc[m].x;
            v[2 * m + 1] = acc64[2 * m + 1] + (double)acc[m].y;
        }
        flush_tile<KB>(red, v, ct0, a);
    }
}

// ---------------------------------------------------------------------------------------
// edge kernel: tiles only partly inside a line's extent, |z|^2 >= Z2 on the whole tile
// ---------------------------------------------------------------------------------------
// Same shape as the mid kernel; the exact integer extent (R7) is applied by selecting the term to zero
// where the lane's bin lies outside [ilo, ihi] (two compares and a select on the ALU pipe).
constexpr int kSubE = 512;
constexpr int kLPTE = kSubE / kThreads;

template <int KB>
__global__ void __launch_bounds__(kThreads, 4) edge_kernel(AccArgs a)
{
    constexpr int kTB = 32 * KB;
    constexpr int M = KB / 2;
    static_assert(sizeof(double) * kWarps * kTB <= sizeof(float4) * 2 * kSubE, "red must fit in the staging buffers");
    __shared__ float4 sm[2][kSubE];       // { -tl, G2, c, 1.5 a2 }
    __shared__ float2 sm2[2][kSubE];      // { ilo, ihi } relative to the tile
    __shared__ int s_unit;
    double* red = reinterpret_cast<double*>(&sm[0][0]);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int32_t* __restrict__ prefix = a.prefix_edge;
    const int base = prefix[0], total = prefix[a.n_ct];

    float2 tb[M];
#pragma unroll
    for (int m = 0; m < M; ++m) {
        float b0 = (float)(lane + 64 * m);
        tb[m] = make_float2(b0, b0 + 32.0f);
    }

    for (;;) {
        const int u = next_unit(&a.st->unit_counter_edge, &s_unit) + base;
        if (u >= total) break;
        const int ct = find_tile(prefix, a.n_ct, u);
        const int64_t ct0 = (int64_t)ct * kTB;
        const TileRange r = a.tr[ct];
        const int sl0 = r.A0, sl1 = r.EL, sr0 = r.ER, sr1 = r.A1;
        const int v_lo = (u - prefix[ct]) * a.chunk;
        const int v_hi = min(v_lo + a.chunk, (sl1 - sl0) + (sr1 - sr0));
        const int l0 = min(sl0 + v_lo, sl1), l1 = min(sl0 + v_hi, sl1);
        const int r0 = sr0 + max(v_lo - (sl1 - sl0), 0), r1 = sr0 + max(v_hi - (sl1 - sl0), 0);
        const int nl = l1 - l0, nt = nl + (r1 - r0);
        if (nt <= 0) continue;
        if (threadIdx.x == 0) atomicAdd(&a.st->units_edge, 1ULL);

        float2 acc[M];
        double acc64[KB];
#pragma unroll
        for (int m = 0; m < M; ++m) acc[m] = make_float2(0.f, 0.f);
#pragma unroll
        for (int j = 0; j < KB; ++j) acc64[j] = 0.0;
        int since_flush = 0;

        float4 preA[kLPTE], preB[kLPTE];
        auto fetch = [&](int v0) {
#pragma unroll
            for (int k = 0; k < kLPTE; ++k) {
                const int v = v0 + threadIdx.x + k * kThreads;
                if (v < nt) {
                    const int li = v < nl ? l0 + v : r0 + (v - nl);
                    preA[k] = a.recA[li];
                    preB[k] = a.recB[li];
                }
            }
        };
        auto stash = [&](int v0, int buf) {
#pragma unroll
            for (int k = 0; k < kLPTE; ++k) {
                const int i = threadIdx.x + k * kThreads;
                if (v0 + i < nt) {
                    const int64_t lim = 1 << 24;
                    const float tl = (float)((int64_t)__float_as_int(preA[k].x) - ct0) + preA[k].y;
                    int64_t dlo = (int64_t)__float_as_int(preB[k].y) - ct0, dhi = (int64_t)__float_as_int(preB[k].z) - ct0;
                    dlo = max(-lim, min(lim, dlo));
                    dhi = max(-lim, min(lim, dhi));
                    sm[buf][i] = make_float4(-tl, preA[k].z, preA[k].w, 1.5f * preB[k].x);
                    sm2[buf][i] = make_float2((float)dlo, (float)dhi);
                }
            }
        };
        fetch(0);
        stash(0, 0);
        __syncthreads();
        int buf = 0;
        for (int v0 = 0; v0 < nt; v0 += kSubE, buf ^= 1) {
            const bool more = v0 + kSubE < nt;
            if (more) fetch(v0 + kSubE);
            const float4* __restrict__ smb = sm[buf];
            const float2* __restrict__ smm = sm2[buf];
            int l, le;
            warp_share(min(kSubE, nt - v0), warp, l, le);
            while (l < le) {
                const int stop = min(le, l + (kFlush - since_flush));
                since_flush += stop - l;
                for (; l < stop; ++l) {
                    const float4 r1 = smb[l];
                    const float2 ext = smm[l];
                    const float2 n1 = bcast2(r1.x), g1 = bcast2(r1.y), c1 = bcast2(r1.z);
                    const float2 A1 = bcast2(r1.w), one = bcast2(1.0f);
                    const float2 nA2 = bcast2(-1.33333333f * r1.w * r1.y);
#pragma unroll
                    for (int m = 0; m < M; ++m) {
                        const float2 t1 = __fadd2_rn(tb[m], n1);
                        const float2 q1 = __ffma2_rn(t1, t1, g1);
                        const float2 rr = rcp2(q1);
                        const float2 uu = __ffma2_rn(nA2, rr, A1);
                        const float2 vv = __ffma2_rn(uu, rr, one);
                        float2 ww = __fmul2_rn(rr, vv);
                        ww.x = (tb[m].x >= ext.x && tb[m].x <= ext.y) ? ww.x : 0.f;     // exact integer extent (R7)
                        ww.y = (tb[m].y >= ext.x && tb[m].y <= ext.y) ? ww.y : 0.f;
                        acc[m] = __ffma2_rn(c1, ww, acc[m]);
                    }
                }
                if (since_flush >= kFlush) {
#pragma unroll
                    for (int m = 0; m < M; ++m) {
                        acc64[2 * m] += (double)acc[m].x;
                        acc64[2 * m + 1] += (double)acc[m].y;
                        acc[m] = make_float2(0.f, 0.f);
                    }
                    since_flush = 0;
                }
            }
            if (more) stash(v0 + kSubE, buf ^ 1);
            __syncthreads();
        }
        double v[KB];
#pragma unroll
        for (int m = 0; m < M; ++m) {
            v[2 * m] = acc64[2 * m] + (double)acc[m].x;
            v[2 * m + 1] = acc64[2 * m + 1] + (double)acc[m].y;
        }
        flush_tile<KB>(red, v, ct0, a);
    }
}

constexpr int kNodeCtas = kP <= 8 ? 6 : 4;   // resident CTAs per SM of the node kernel (register budget grows with the node count)

}  // namespace hk
#include "hk_centre.cuh"               // the line centres: centre_row_kernel, centre_lane_kernel
namespace hk {

// ---------------------------------------------------------------------------------------
// near / edge kernel
// ---------------------------------------------------------------------------------------
constexpr int kSubN = 512;             // lines per staged batch
constexpr int kLPTN = kSubN / kThreads;
constexpr float kWideCore = 64.0f;     // (core half-width in bins)^2 from which the core is evaluated in the row pass
// per-line flags, decided once per (line, tile) when the line is staged
constexpr int kFlagFull = 1;           // the whole tile is inside the extent: no mask
constexpr int kFlagNoCore = 2;         // |z|^2 >= Z2 on every bin of the tile
constexpr int kFlagFar = 4;            // |z|^2 >= Z1 on every bin of the tile: one term is enough
constexpr int kFlagWide = 8;           // core spans >= 16 bins: evaluated in the row pass

// One line against the warp's KB rows of 32 bins.  A = { jc - ct0, f, G2, c }, B = { A1, -A2 (binned Gaussian: the low
// part of f), qc, cK }, C = { ilo - ct0, ihi - ct0, y (binned Gaussian: dnu/alpha_D), flags }.
template <int KB, bool kTwoTerm, bool kMask, bool kCore>
__device__ __forceinline__ void near_rows(float2 (&acc)[KB / 2], const float2 (&tb)[KB / 2], const float4 A,
                                          const float4 B, const float4 C, const bool wide, const int profile = 0)
{
    const float2 ndl = bcast2(-A.x), nf = bcast2(-A.y), g = bcast2(A.z);
    const float2 A1 = bcast2(B.x), nA2 = bcast2(B.y), one = bcast2(1.0f);
    const float2 c = bcast2(A.w);
    const float qc = B.z, lo = C.x, hi = C.y;
    const bool binned = profile == HK_PROFILE_BINNED_GAUSSIAN;
    float inv_a = 0.f;
    if (kCore && wide) inv_a = binned ? C.z : sqrtf(HK_Z2 / qc);
#pragma unroll
    for (int m = 0; m < KB / 2; ++m) {
        const float2 d = __fadd2_rn(tb[m], ndl);            // exact: both are small integers
        const float2 t = __fadd2_rn(d, nf);
        const float2 q = __ffma2_rn(t, t, g);
        const float2 rr = rcp2(q);
        float2 ww = rr;
        if (kTwoTerm) {
            const float2 uu = __ffma2_rn(nA2, rr, A1);
            const float2 vv = __ffma2_rn(uu, rr, one);
            ww = __fmul2_rn(rr, vv);
        }
        bool in0 = true, in1 = true, co0 = false, co1 = false;
        if (kMask) {                                         // exact integer extent (R7)
            in0 = (tb[m].x >= lo) && (tb[m].x <= hi);
            in1 = (tb[m].y >= lo) && (tb[m].y <= hi);
        }
        if (kCore) { co0 = q.x < qc; co1 = q.y < qc; }
        // selected, not multiplied by a zero amplitude: 1/q at q = 0 (a zero-width line on a grid point) is not finite
        if (kMask || kCore) {
            ww.x = (in0 && !co0) ? ww.x : 0.f;
            ww.y = (in1 && !co1) ? ww.y : 0.f;
        }
        acc[m] = __ffma2_rn(c, ww, acc[m]);
        if (kCore && wide) {
            const float flo = binned ? B.y : 0.f;
            if (__any_sync(0xffffffffu, in0 && co0)) {
                if (in0 && co0) acc[m].x += core_term(profile, B.w, d.x, A.y, flo, inv_a, C.z);
            }
            if (__any_sync(0xffffffffu, in1 && co1)) {
                if (in1 && co1) acc[m].y += core_term(profile, B.w, d.y, A.y, flo, inv_a, C.z);
            }
        }
    }
}

template <int KB>
__global__ void __launch_bounds__(kThreads, 2) near_kernel(AccArgs a)
{
    constexpr int kTB = 32 * KB;
    constexpr int M = KB / 2;
    static_assert(sizeof(double) * kWarps * kTB <= sizeof(float4) * 2 * kSubN, "red must fit in smA + smB");
    __shared__ float4 smem[3][kSubN];          // A, B, C records (see near_rows)
    __shared__ float sacc[kWarps][kTB];        // per-warp bin tile of the lane pass
    __shared__ int s_unit;
    float4* smA = smem[0];
    float4* smB = smem[1];
    float4* smC = smem[2];
    double* red = reinterpret_cast<double*>(&smem[0][0]);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int32_t* __restrict__ prefix = a.prefix_near;
    const int base = prefix[0], total = prefix[a.n_ct];
    const float whi = (float)(kTB - 1);

    float2 tb[M];
#pragma unroll
    for (int m = 0; m < M; ++m) {
        float b0 = (float)(lane + 64 * m);
        tb[m] = make_float2(b0, b0 + 32.0f);
    }
#pragma unroll
    for (int j = 0; j < KB; ++j) sacc[warp][lane + 32 * j] = 0.f;

    for (;;) {
        const int u = next_unit(&a.st->unit_counter_near, &s_unit) + base;
        if (u >= total) break;
        const int ct = find_tile(prefix, a.n_ct, u);
        const int64_t ct0 = (int64_t)ct * kTB;
        const TileRange r = a.tr[ct];
        // the generic parts of the edge and centre segments walked as one list; this unit takes lines [v_lo, v_hi) of it
        const int s0 = r.FL0 - r.EL, s1 = r.CL - r.ML1, s2 = r.MR0 - r.CR, s3 = r.ER - r.FR1;
        const int v_lo = (u - prefix[ct]) * a.chunk;
        const int v_hi = min(v_lo + a.chunk, s0 + s1 + s2 + s3);
        auto clip = [](int v, int n) { return max(0, min(v, n)); };
        const int g0 = r.EL + clip(v_lo, s0), n0 = clip(v_hi, s0) - clip(v_lo, s0);
        const int g1 = r.ML1 + clip(v_lo - s0, s1), n1 = clip(v_hi - s0, s1) - clip(v_lo - s0, s1);
        const int g2 = r.CR + clip(v_lo - s0 - s1, s2), n2 = clip(v_hi - s0 - s1, s2) - clip(v_lo - s0 - s1, s2);
        const int g3 = r.FR1 + clip(v_lo - s0 - s1 - s2, s3), n3 = clip(v_hi - s0 - s1 - s2, s3) - clip(v_lo - s0 - s1 - s2, s3);
        const int nt = n0 + n1 + n2 + n3;
        if (nt <= 0) continue;
        if (threadIdx.x == 0) atomicAdd(&a.st->units_near, 1ULL);

        float2 acc[M];
        double acc64[KB];
#pragma unroll
        for (int m = 0; m < M; ++m) acc[m] = make_float2(0.f, 0.f);
#pragma unroll
        for (int j = 0; j < KB; ++j) acc64[j] = 0.0;
        int since_flush = 0;
        auto flush = [&]() {
            __syncwarp();
#pragma unroll
            for (int m = 0; m < M; ++m) {
                acc64[2 * m] += (double)acc[m].x + (double)sacc[warp][lane + 64 * m];
                acc64[2 * m + 1] += (double)acc[m].y + (double)sacc[warp][lane + 64 * m + 32];
                acc[m] = make_float2(0.f, 0.f);
                sacc[warp][lane + 64 * m] = 0.f;
                sacc[warp][lane + 64 * m + 32] = 0.f;
            }
            since_flush = 0;
            __syncwarp();
        };

        float4 preA[kLPTN], preB[kLPTN];
        auto fetch = [&](int v0) {
#pragma unroll
            for (int k = 0; k < kLPTN; ++k) {
                const int v = v0 + threadIdx.x + k * kThreads;
                if (v < nt) {
                    const int li = v < n0 ? g0 + v
                                 : v < n0 + n1 ? g1 + (v - n0)
                                 : v < n0 + n1 + n2 ? g2 + (v - n0 - n1) : g3 + (v - n0 - n1 - n2);
                    preA[k] = a.recA[li];
                    preB[k] = a.recB[li];
                }
            }
        };
        auto stash = [&](int v0) {
#pragma unroll
            for (int k = 0; k < kLPTN; ++k) {
                const int i = threadIdx.x + k * kThreads;
                if (v0 + i < nt) {
                    const float4 ra = preA[k], rb = preB[k];
                    const int64_t lim = 1 << 24;
                    const int64_t dj = (int64_t)__float_as_int(ra.x) - ct0;
                    int64_t dlo = (int64_t)__float_as_int(rb.y) - ct0, dhi = (int64_t)__float_as_int(rb.z) - ct0;
                    dlo = max(-lim, min(lim, dlo));
                    dhi = max(-lim, min(lim, dhi));
                    const float fdj = (float)dj, flo = (float)dlo, fhi = (float)dhi;
                    const bool binned = a.profile == HK_PROFILE_BINNED_GAUSSIAN;
                    const float G2 = binned ? 0.f : ra.z, a2 = rb.x;          // (binned: A.z carries the low part of f)
                    const float qc = binned ? binned_ql(a2) : HK_Z2 * a2;
                    // smallest q = t^2 + G2 over the tile's bins, from below
                    const float pos = fdj + ra.y;
                    const float dist = fmaxf(fmaxf(-pos, pos - whi), 0.f) * 0.999f;
                    const float qmin = fmaf(dist, dist, G2) * 0.9999f;
                    int flags = 0;
                    if (flo <= 0.f && fhi >= whi) flags |= kFlagFull;
                    if (qmin >= qc) flags |= kFlagNoCore;
                    if (qmin >= fmaxf(HK_Z1 * a2, qc)) flags |= kFlagFar;
                    if ((qc - G2) >= kWideCore) flags |= kFlagWide;
                    smA[i] = make_float4(fdj, ra.y, G2, ra.w);
                    smB[i] = make_float4(1.5f * a2, binned ? ra.z : -2.0f * a2 * G2, qc, rb.w);
                    // C.z: y for the Voigt evaluators; the binned Gaussian needs 1/a instead (its y is 0)
                    smC[i] = make_float4(flo, fhi, binned ? sqrtf(1.0f / a2) : sqrtf(G2 / a2), __int_as_float(flags));
                }
            }
        };
        fetch(0);
        for (int v0 = 0; v0 < nt; v0 += kSubN) {
            __syncthreads();                        // previous batch fully consumed
            stash(v0);
            __syncthreads();
            if (v0 + kSubN < nt) fetch(v0 + kSubN);
            int wl0, wl1;
            warp_share(min(kSubN, nt - v0), warp, wl0, wl1);
            // ---- row pass: lanes own bins, the warp walks its lines
#pragma unroll 1
            for (int l = wl0; l < wl1; ++l) {
                const float4 A = smA[l], B = smB[l], C = smC[l];
                const int flags = __float_as_int(C.w);
                if (flags & kFlagFar) {
                    if (flags & kFlagFull) near_rows<KB, false, false, false>(acc, tb, A, B, C, false);
                    else near_rows<KB, false, true, false>(acc, tb, A, B, C, false);
                } else if (flags & kFlagNoCore) {
                    if (flags & kFlagFull) near_rows<KB, true, false, false>(acc, tb, A, B, C, false);
                    else near_rows<KB, true, true, false>(acc, tb, A, B, C, false);
                } else {
                    near_rows<KB, true, true, true>(acc, tb, A, B, C, (flags & kFlagWide) != 0, a.profile);
                }
                if (++since_flush >= kFlush) flush();
            }
            // ---- lane pass: lane <-> line, each lane walks its line's narrow core (|z|^2 < Z2) inside this tile
#pragma unroll 1
            for (int lb = wl0; lb < wl1; lb += 32) {
                const int l = lb + lane;
                float dlt = 0.f, f = 0.f, flo = 0.f, G2 = 0.f, cK = 0.f, qc = 0.f, y = 0.f;
                int cnt = 0;
                float clo = 0.f;
                if (l < wl1) {
                    const float4 A = smA[l], B = smB[l], C = smC[l];
                    const int flags = __float_as_int(C.w);
                    if (!(flags & (kFlagNoCore | kFlagWide))) {
                        dlt = A.x; f = A.y; G2 = A.z; cK = B.w; qc = B.z; y = C.z;
                        if (a.profile == HK_PROFILE_BINNED_GAUSSIAN) flo = B.y;
                        const float h2 = qc - G2;
                        const float hw = sqrtf(fmaxf(h2, 0.f)) + 1.0f;           // |t| < hw covers every q < qc
                        const float pos = dlt + f;
                        clo = fmaxf(fmaxf(ceilf(pos - hw), C.x), 0.f);
                        const float chi = fminf(fminf(floorf(pos + hw), C.y), whi);
                        if (h2 > 0.f && chi >= clo) cnt = (int)(chi - clo) + 1;
                    }
                }
                int maxcnt = cnt;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) maxcnt = max(maxcnt, __shfl_xor_sync(0xffffffffu, maxcnt, o));
                if (maxcnt == 0) continue;
                const float inv_a = a.profile == HK_PROFILE_BINNED_GAUSSIAN ? y : sqrtf(HK_Z2 / fmaxf(qc, 1e-30f));
                for (int o = 0; o < maxcnt; ++o) {
                    float val = 0.f;
                    int bin = -1;
                    if (o < cnt) {
                        const float fb = clo + (float)o;
                        const float d = fb - dlt;
                        const float t = d - f;
                        const float q = fmaf(t, t, G2);
                        if (q < qc) { val = core_term(a.profile, cK, d, f, flo, inv_a, y); bin = (int)fb; }
                    }
                    // combine equal bins in the warp (sorted lines: neighbours share bins), one add per distinct bin
                    unsigned todo = __ballot_sync(0xffffffffu, bin >= 0);
                    while (todo) {
                        const int leader = __ffs(todo) - 1;
                        const int b = __shfl_sync(0xffffffffu, bin, leader);
                        const bool mine = (bin == b);
                        float sum = mine ? val : 0.f;
#pragma unroll
                        for (int x = 16; x > 0; x >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, x);
                        if (lane == leader) sacc[warp][b] += sum;
                        todo &= ~__ballot_sync(0xffffffffu, mine);
                    }
                }
                since_flush += 32;     // the tile holds at most 32 lines' terms per bin per pass
                if (since_flush >= kFlush) flush();
            }
        }
        flush();
        __syncthreads();               // every warp is done with the staging buffers: red may overwrite them
        flush_tile<KB>(red, acc64, ct0, a);
    }
}

// ---------------------------------------------------------------------------------------
// node kernel: separated (line, tile) pairs evaluated at the tile's kP Chebyshev nodes
// ---------------------------------------------------------------------------------------
// Lanes walk LINES (one line per lane, coalesced 16 B records), every lane holds the tile's kP node
// positions and kP partial sums in registers; two nodes share one reciprocal.  The partial sums are
// combined with warp shuffles, then across warps, and reach the (level, tile) node sums with one
// fp64 atomic per node per work unit.  Formula: two asymptotic terms (valid: |z|^2 >= Z2 on the tile).
__global__ void __launch_bounds__(kThreads, kNodeCtas) node_kernel(AccArgs a)
{
    constexpr int M = kP / 2;
    __shared__ float red[kWarps][kP];
    __shared__ int s_unit;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int32_t* __restrict__ prefix = a.prefix_node;
    const int n_e = a.lv.n_entries;
    const int base = prefix[0], total = prefix[n_e];
    for (;;) {
        const int u = next_unit(&a.st->unit_counter_node, &s_unit) + base;
        if (u >= total) break;
        const int e = find_tile(prefix, n_e, u);
        int l = 0;
        while (l + 1 < a.lv.n_levels && e >= a.lv.off[l + 1]) ++l;
        const int64_t W = (int64_t)a.lv.w0 << l;
        const int64_t tile0 = (int64_t)(e - a.lv.off[l]) * W;
        const NodeRange r = a.nr[e];
        const int s0 = r.a1 - r.a0, s1 = r.b1 - r.b0, s2 = r.c1 - r.c0, s3 = r.d1 - r.d0;
        const int v_lo = (u - prefix[e]) * a.chunk_node;
        const int v_hi = min(v_lo + a.chunk_node, s0 + s1 + s2 + s3);
        if (v_hi <= v_lo) continue;
        if (threadIdx.x == 0) atomicAdd(&a.st->units_node, 1ULL);
        float2 xk[M], acc[M];
        const double hc = 0.5 * (double)(W - 1), hw = 0.5 * (double)W;
#pragma unroll
        for (int m = 0; m < M; ++m) {
            xk[m] = make_float2((float)(hc + hw * kChebX[2 * m]), (float)(hc + hw * kChebX[2 * m + 1]));
            acc[m] = make_float2(0.f, 0.f);
        }
        for (int v0 = v_lo + 32 * warp; v0 < v_hi; v0 += kThreads) {        // (warp-uniform trip count)
            const int v = v0 + lane;
            const bool live = v < v_hi;
            const int li = v < s0 ? r.a0 + v
                         : v < s0 + s1 ? r.b0 + (v - s0)
                         : v < s0 + s1 + s2 ? r.c0 + (v - s0 - s1) : r.d0 + (v - s0 - s1 - s2);
            float4 rec = make_float4(0.f, 0.f, 1.f, 0.f);
            if (live) rec = a.recN[li];
            const uint32_t pk = (uint32_t)__float_as_int(rec.y);
            const float f = (float)(pk >> 19) * (1.0f / 8192.0f);
            const float npos = -((float)((int64_t)__float_as_int(rec.x) - tile0) + f);
            const float2 np2 = bcast2(npos), g2 = bcast2(rec.z), c2 = bcast2(rec.w);
            // far from the tile (|z|^2 >= Z1 on all of it: a prefix of the left lists, a suffix of the right ones): the
            // Lorentzian alone.  The lines of a warp are neighbours in the sorted order, so a warp is almost always all far
            // or all near; in a mixed warp the far lines run the two-term form with a^2 = 0, which is the same value bit
            // for bit -- what a (line, tile) pair contributes never depends on its neighbours
            const bool far = !live || li < r.fL || li >= r.fR;
            if (__all_sync(0xffffffffu, far)) {
#pragma unroll
                for (int m = 0; m < M; ++m) {
                    const float2 t = __fadd2_rn(xk[m], np2);
                    const float2 q = __ffma2_rn(t, t, g2);
                    const float R = rcp_approx(q.x * q.y);             // 1/q.x = R q.y, 1/q.y = R q.x
                    acc[m] = __ffma2_rn(c2, make_float2(R * q.y, R * q.x), acc[m]);
                }
            } else {
                const float a2 = far ? 0.f : __int_as_float((int)((pk & 0x7FFFFu) << 12));
                const float2 one = bcast2(1.0f), A1 = bcast2(1.5f * a2), nA2 = bcast2(-2.0f * a2 * rec.z);
#pragma unroll
                for (int m = 0; m < M; ++m) {
                    const float2 t = __fadd2_rn(xk[m], np2);
                    const float2 q = __ffma2_rn(t, t, g2);
                    const float R = rcp_approx(q.x * q.y);             // 1/q.x = R q.y, 1/q.y = R q.x
                    const float2 rr = make_float2(R * q.y, R * q.x);
                    const float2 uu = __ffma2_rn(nA2, rr, A1);
                    const float2 vv = __ffma2_rn(uu, rr, one);
                    const float2 ww = __fmul2_rn(rr, vv);
                    acc[m] = __ffma2_rn(c2, ww, acc[m]);
                }
            }
        }
#pragma unroll
        for (int m = 0; m < M; ++m) {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                acc[m].x += __shfl_xor_sync(0xffffffffu, acc[m].x, o);
                acc[m].y += __shfl_xor_sync(0xffffffffu, acc[m].y, o);
            }
        }
        if (lane == 0) {
#pragma unroll
            for (int m = 0; m < M; ++m) { red[warp][2 * m] = acc[m].x; red[warp][2 * m + 1] = acc[m].y; }
        }
        __syncthreads();
        if (threadIdx.x < kP) {
            double sum = 0.0;
#pragma unroll
            for (int w = 0; w < kWarps; ++w) sum += (double)red[w][threadIdx.x];
            if (sum != 0.0) atomicAdd(a.node_acc + (size_t)e * kP + threadIdx.x, sum);
        }
    }
}

// ---------------------------------------------------------------------------------------
// edge-node kernel: extent ends in separated tiles, evaluated at the tile's kP nodes (edge_keys, hk_preprocess.cuh)
// ---------------------------------------------------------------------------------------
// Lanes walk the sorted LINES.  For each end of its extent a lane finds the level-0 tile the end falls in, evaluates
// its line at that tile's nodes (two-term asymptotic, as node_kernel) and adds the kP values to the accumulators of
// the bin where the extent ends: side 0 = last bin ihi (the line covers the bins <= ihi of the tile), side 1 = first
// bin ilo (bins >= ilo).  Neighbouring lines end in the same few bins, so equal bins are summed in the warp first and
// one lane issues the fp64 atomics.  edge_scan_kernel turns the accumulators into suffix (side 0) / prefix (side 1)
// sums over each tile, edge_bins_kernel interpolates them onto the bins.  The sum of interpolants over any subset of
// lines is the interpolant of that subset's node sums, so the per-bin subsets cost nothing extra.
// Sum kP per-lane values over the lanes with `mine` set and add the kP sums to dst[0..kP) (fp64 atomics).
// Transposing reduction: each exchange halves the values a lane carries (8 -> 4 -> 2 -> 1 over lane bits 4, 3, 2), two
// butterfly steps finish bits 1, 0: 9 shuffles instead of 40.  Lane l then holds the sum of value j = (bit4, bit3, bit2
// of l); the lanes with l % 4 == 0 issue one atomic each.  Nodes beyond the first eight (kP = 10, 12) go through a
// second, shorter fold of the same kind.  Called by all 32 lanes.
__device__ __forceinline__ void warp_fold_add(double* __restrict__ dst, const float (&v)[kP], bool mine, int lane)
{
    static_assert(kP == 8 || kP == 10 || kP == 12, "the folds below are written for 8, 10 or 12 nodes");
    float a[8], b4[4], c2[2];
#pragma unroll
    for (int j = 0; j < 8; ++j) a[j] = mine ? v[j] : 0.f;
    const bool h4 = (lane & 16) != 0, h3 = (lane & 8) != 0, h2 = (lane & 4) != 0;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const float send = h4 ? a[j] : a[j + 4], keep = h4 ? a[j + 4] : a[j];
        b4[j] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
    }
#pragma unroll
    for (int j = 0; j < 2; ++j) {
        const float send = h3 ? b4[j] : b4[j + 2], keep = h3 ? b4[j + 2] : b4[j];
        c2[j] = keep + __shfl_xor_sync(0xffffffffu, send, 8);
    }
    float d = (h2 ? c2[1] : c2[0]) + __shfl_xor_sync(0xffffffffu, h2 ? c2[0] : c2[1], 4);
    d += __shfl_xor_sync(0xffffffffu, d, 2);
    d += __shfl_xor_sync(0xffffffffu, d, 1);
    const int j = ((lane >> 4) & 1) * 4 + ((lane >> 3) & 1) * 2 + ((lane >> 2) & 1);
    if ((lane & 3) == 0 && d != 0.f) atomicAdd(dst + j, (double)d);
    if constexpr (kP == 12) {
        // values 8..11: 4 -> 2 -> 1 over lane bits 4, 3, then three butterfly steps; lane l holds j = 8 + (bit4, bit3)
        float e[4], f2[2];
#pragma unroll
        for (int q = 0; q < 4; ++q) e[q] = mine ? v[8 + q] : 0.f;
#pragma unroll
        for (int q = 0; q < 2; ++q) {
            const float send = h4 ? e[q] : e[q + 2], keep = h4 ? e[q + 2] : e[q];
            f2[q] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
        }
        float g = (h3 ? f2[1] : f2[0]) + __shfl_xor_sync(0xffffffffu, h3 ? f2[0] : f2[1], 8);
        g += __shfl_xor_sync(0xffffffffu, g, 4);
        g += __shfl_xor_sync(0xffffffffu, g, 2);
        g += __shfl_xor_sync(0xffffffffu, g, 1);
        const int jj = 8 + ((lane >> 4) & 1) * 2 + ((lane >> 3) & 1);
        if ((lane & 7) == 0 && g != 0.f) atomicAdd(dst + jj, (double)g);
    } else if constexpr (kP == 10) {
        // values 8, 9: 2 -> 1 over lane bit 4, then four butterfly steps; lane l holds j = 8 + bit4
        const float e0 = mine ? v[8] : 0.f, e1 = mine ? v[kP - 1] : 0.f;
        float g = (h4 ? e1 : e0) + __shfl_xor_sync(0xffffffffu, h4 ? e0 : e1, 16);
        g += __shfl_xor_sync(0xffffffffu, g, 8);
        g += __shfl_xor_sync(0xffffffffu, g, 4);
        g += __shfl_xor_sync(0xffffffffu, g, 2);
        g += __shfl_xor_sync(0xffffffffu, g, 1);
        if ((lane & 15) == 0 && g != 0.f) atomicAdd(dst + 8 + ((lane >> 4) & 1), (double)g);
    }
}

__device__ __forceinline__ void warp_add_by_bin(double* __restrict__ acc, int64_t bin, const float (&v)[kP], int lane)
{
    unsigned todo = __ballot_sync(0xffffffffu, bin >= 0);
    while (todo) {
        const int leader = __ffs(todo) - 1;
        const int64_t b = __shfl_sync(0xffffffffu, bin, leader);
        const bool mine = (bin == b);
        const unsigned grp = __ballot_sync(0xffffffffu, mine);
        if (__popc(grp) == 1) {
            if (mine) {
#pragma unroll
                for (int j = 0; j < kP; ++j) atomicAdd(acc + (size_t)b * kP + j, (double)v[j]);
            }
        } else {
            warp_fold_add(acc + (size_t)b * kP, v, mine, lane);
        }
        todo &= ~grp;
    }
}

// ---------------------------------------------------------------------------------------
// node kernel, line-stationary form: a CTA keeps a chunk of consecutive sorted lines in shared memory and walks the
// (level, tile) entries those lines are evaluated at
// ---------------------------------------------------------------------------------------
// node_kernel above is entry-stationary: a work unit is (entry, chunk of its lines), every line record is fetched once
// per entry it belongs to (~19 times) and every unit starts with a search for its entry.  Here the loop order is turned
// round: the records of kNLChunk consecutive lines are staged ONCE (16 B per line), the entries that hold any of them
// are found from the geometry (a generous superset of tiles per level, then the exact index ranges of NodeRange decide
// membership, so every (line, tile) pair is evaluated exactly once, as node_range_kernel counted it), and each warp
// walks those entries with its 512 lines, 16 per lane, before ONE fold + 12 atomics per (warp, entry).
constexpr int kNLChunk = 2048;                    // lines per chunk
constexpr int kNLThreads = 128;                  // threads per CTA: 4 warps of 512 lines
constexpr int kNLCtas = 5;                       // resident CTAs per SM (40 KB of shared memory each)
constexpr int kNLPerLane = kNLChunk / kNLThreads; // lines per lane per entry: amortises the per-(warp, entry) work
constexpr int kNLMaxEnt = kNLThreads;            // entries resolved per round (one candidate per thread)

struct __align__(16) NLEntry {
    NodeRange r;
    int32_t e, l;
    int32_t D;           // (centre bin of the chunk's first line) - (first bin of the tile)
    int32_t pad;
};
constexpr size_t kNLSmemBytes = sizeof(float4) * kNLChunk + sizeof(NLEntry) * kNLMaxEnt;

// tile-index intervals [lo[i], hi[i]] (i < 3, disjoint, possibly empty) of level l that can hold lines with centre bins
// in [jlo, jhi]; a superset -- membership is decided by NodeRange
__device__ __forceinline__ void nl_candidates(const Params& p, const Levels& lv, int l, int64_t jlo, int64_t jhi,
                                               int64_t (&lo)[3], int64_t (&hi)[3])
{
    const int64_t W = (int64_t)lv.w0 << l;
    const int64_t nt = lv.off[l + 1] - lv.off[l];
    const bool top = l + 1 == lv.n_levels;
    auto tdiv = [&](int64_t b) { return b >= 0 ? b / W : -((-b + W - 1) / W); };     // floor(b / W)
    for (int i = 0; i < 3; ++i) { lo[i] = 0; hi[i] = -1; }
    // lines the parent does not take: closer than the parent's separation, or inside the core bound of the parent tile
    double rc = 1.0e18;
    if (p.kappa2 < 0.9) rc = p.kappa2 * (p.numin_bins + (double)jhi + 2.0) / (1.0 - p.kappa2) + 8.0;
    const double ra_d = fmax((p.sep + 0.5) * (double)W, rc + 1.5 * (double)W) + (double)W + 8.0;
    const int64_t big = (int64_t)1 << 40;
    const int64_t RA = ra_d < (double)big ? (int64_t)ra_d : big;
    if (p.uncut) {
        if (top || RA >= big) { lo[0] = 0; hi[0] = nt - 1; }
        else { lo[0] = tdiv(jlo - RA); hi[0] = tdiv(jhi + RA); }
    } else {
        const int64_t reach = p.cb_ceil + W + 8;
        if (top || 2 * reach / W <= 40 || RA >= reach) { lo[0] = tdiv(jlo - reach); hi[0] = tdiv(jhi + reach); }
        else {
            // left extent end (the parent tile is not inside the extent, the child is), centre, right extent end
            lo[0] = tdiv(jlo - p.cb_ceil - W - 8); hi[0] = tdiv(jhi - p.cb_floor + 2 * W + 8);
            lo[1] = tdiv(jlo - RA);                hi[1] = tdiv(jhi + RA);
            lo[2] = tdiv(jlo + p.cb_floor - 2 * W - 8); hi[2] = tdiv(jhi + p.cb_ceil + W + 8);
        }
    }
    int64_t prev = -1;
    for (int i = 0; i < 3; ++i) {                 // clip to the level, make disjoint (they are ordered left to right)
        lo[i] = max(lo[i], max((int64_t)0, prev + 1));
        hi[i] = min(hi[i], nt - 1);
        if (hi[i] >= lo[i]) prev = hi[i];
    }
}

constexpr int kNLDirect = 3;      // node pairs (of kP / 2) whose two reciprocals are taken directly instead of through their product
__global__ void __launch_bounds__(kNLThreads, kNLCtas) node_lines_kernel(Params p, AccArgs a)
{
    constexpr int M = kP / 2;
    extern __shared__ __align__(16) unsigned char nl_smem[];      // kNLSmemBytes, opted in by the host (> 48 KB)
    float4* sRec = reinterpret_cast<float4*>(nl_smem);            // [kNLChunk] recN with the centre bin relative to the chunk's first
    NLEntry* sEnt = reinterpret_cast<NLEntry*>(nl_smem + sizeof(float4) * kNLChunk);   // [kNLMaxEnt]
    __shared__ float sXk[kMaxLevels][kP];         // node positions of a tile of each level, relative to its first bin
    __shared__ int64_t sLo[kMaxLevels][3], sHi[kMaxLevels][3];
    __shared__ int sCnt[kMaxLevels + 1];          // candidates before level l
    __shared__ int s_nent;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const Levels& lv = a.lv;
    apply_shift_bound(p, a.st);
    for (int i = threadIdx.x; i < lv.n_levels * kP; i += kNLThreads) {
        const int l = i / kP, k = i - l * kP;
        const int64_t W = (int64_t)lv.w0 << l;
        sXk[l][k] = (float)(0.5 * (double)(W - 1) + 0.5 * (double)W * kChebX[k]);
    }
    const int n_act = a.st->n_act;
    const int n_chunks = (n_act + kNLChunk - 1) / kNLChunk;
    unsigned long long n_eval = 0;                // (line, tile) pairs this thread evaluated
    for (int chunk = blockIdx.x; chunk < n_chunks; chunk += gridDim.x) {
        const int c_lo = chunk * kNLChunk, c_hi = min(c_lo + kNLChunk, n_act);
        const int64_t jc0 = __float_as_int(a.recN[c_lo].x), jc1 = __float_as_int(a.recN[c_hi - 1].x);
        __syncthreads();                          // the previous chunk is done with the shared arrays
#pragma unroll
        for (int k = 0; k < kNLPerLane; ++k) {
            const int i = threadIdx.x + k * kNLThreads;
            float4 o = make_float4(0.f, 0.f, 1.f, 0.f);
            if (c_lo + i < c_hi) {
                o = a.recN[c_lo + i];
                o.x = __int_as_float((int)((int64_t)__float_as_int(o.x) - jc0));      // (fits: the list is sorted, |jc| < 2^30)
            }
            sRec[i] = o;
        }
        if (threadIdx.x < lv.n_levels) {
            int64_t lo[3], hi[3];
            nl_candidates(p, lv, threadIdx.x, jc0, jc1, lo, hi);
            for (int i = 0; i < 3; ++i) { sLo[threadIdx.x][i] = lo[i]; sHi[threadIdx.x][i] = hi[i]; }
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            int tot = 0;
            for (int l = 0; l < lv.n_levels; ++l) {
                sCnt[l] = tot;
                for (int i = 0; i < 3; ++i) tot += (int)max((int64_t)0, sHi[l][i] - sLo[l][i] + 1);
            }
            sCnt[lv.n_levels] = tot;
        }
        __syncthreads();
        const int n_cand = sCnt[lv.n_levels];
        for (int round0 = 0; round0 < n_cand; round0 += kNLMaxEnt) {
            if (threadIdx.x == 0) s_nent = 0;
            __syncthreads();
            const int ci = round0 + threadIdx.x;
            if (ci < n_cand) {
                int l = 0;
                while (l + 1 < lv.n_levels && ci >= sCnt[l + 1]) ++l;
                int64_t off = ci - sCnt[l], j = -1;
                for (int i = 0; i < 3 && j < 0; ++i) {
                    const int64_t c = max((int64_t)0, sHi[l][i] - sLo[l][i] + 1);
                    if (off < c) j = sLo[l][i] + off; else off -= c;
                }
                const int e = lv.off[l] + (int)j;
                const NodeRange r = a.nr[e];
                auto ov = [&](int x0, int x1) { return x1 > x0 && x0 < c_hi && x1 > c_lo; };
                if (ov(r.a0, r.a1) || ov(r.b0, r.b1) || ov(r.c0, r.c1) || ov(r.d0, r.d1)) {
                    const int slot = atomicAdd(&s_nent, 1);
                    NLEntry E;
                    E.r = r; E.e = e; E.l = l; E.pad = 0;
                    E.D = (int32_t)(jc0 - j * ((int64_t)lv.w0 << l));           // |.| < 2^31: both lie within 2^30 bins of the grid
                    sEnt[slot] = E;
                }
            }
            __syncthreads();
            const int nent = s_nent;
            const int wl = c_lo + warp * (32 * kNLPerLane), wh = min(wl + 32 * kNLPerLane, c_hi);
            for (int ei = 0; ei < nent; ++ei) {
                const NodeRange r = sEnt[ei].r;
                auto ovw = [&](int x0, int x1) { return x1 > x0 && x0 < wh && x1 > wl; };
                if (!(ovw(r.a0, r.a1) || ovw(r.b0, r.b1) || ovw(r.c0, r.c1) || ovw(r.d0, r.d1))) continue;   // (warp-uniform)
                const int l = sEnt[ei].l;
                const int D = sEnt[ei].D;
                float2 xk[M], acc[M];
#pragma unroll
                for (int m = 0; m < M; ++m) {
                    xk[m] = make_float2(sXk[l][2 * m], sXk[l][2 * m + 1]);
                    acc[m] = make_float2(0.f, 0.f);
                }
                const float4* __restrict__ wrec = sRec + warp * (32 * kNLPerLane);
                const int fLr = r.fL - wl, fRr = r.fR - wl;        // far boundaries relative to the warp's first line
                const int gLr = r.gL - wl, gRr = r.gR - wl;        // core boundaries (empty unless core_nodes)
                // the members among this warp's lines: up to four runs [s, e) of offsets (one, in dense lists); every
                // bound below is warp-uniform, the lanes only compare their own offset with it
                auto run = [&](int x0, int x1) {
                    const int s_ = max(x0, wl) - wl, e_ = min(x1, wh) - wl;
                    if (e_ <= s_) return;
                    if (lane == 0) n_eval += (unsigned)(e_ - s_);
                    // far from the tile (|z|^2 >= Z1 on all of it): the Lorentzian alone; a mixed warp runs the two-term
                    // form with a^2 = 0 for its far lines, which is the same value bit for bit
                    const bool all_far = e_ <= fLr || s_ >= fRr, none_far = s_ >= fLr && e_ <= fRr;
#pragma unroll 1
                    for (int o0 = s_ & ~31; o0 < e_; o0 += 32) {
                        const int o = o0 + lane;
                        const bool member = o >= s_ && o < e_;
                        const float4 rec = wrec[o];
                        const uint32_t pk = (uint32_t)__float_as_int(rec.y);
                        const float f = (float)(pk >> 19) * (1.0f / 8192.0f);
                        const float2 np2 = bcast2(-((float)(__float_as_int(rec.x) + D) + f)), g2 = bcast2(rec.z);
                        // the core at nodes: lines whose core may reach this tile take the 4-point Gauss-Hermite form
                        // K = y N(X, Y) / D(X, Y), X = t^2 / a^2, Y = G^2 / a^2, amplitude cK y = c sqrt(pi) / a^2; the other
                        // lanes of the batch (amplitude 0, X = 0) follow with the asymptotic forms below
                        const bool core = member && o >= gLr && o < gRr;
                        if (__any_sync(0xffffffffu, core)) {
                            const float a2c = __int_as_float((int)((pk & 0x7FFFFu) << 12));
                            const float ia = (core && a2c > 0.f) ? __fdividef(1.0f, a2c) : 0.f;
                            float n4[3], d4[4];
                            gh4_coeffs(rec.z * ia, n4, d4);
                            const float2 ia2 = bcast2(ia), amp = bcast2(core ? rec.w * 1.7724538509f * ia : 0.f);
#pragma unroll
                            for (int m = 0; m < M; ++m) {
                                const float2 t = __fadd2_rn(xk[m], np2);
                                const float2 X = __fmul2_rn(__fmul2_rn(t, t), ia2);
                                float2 N = __ffma2_rn(bcast2(kGhN), X, bcast2(n4[2]));
                                N = __ffma2_rn(N, X, bcast2(n4[1]));
                                N = __ffma2_rn(N, X, bcast2(n4[0]));
                                float2 Dn = __fadd2_rn(X, bcast2(d4[3]));
                                Dn = __ffma2_rn(Dn, X, bcast2(d4[2]));
                                Dn = __ffma2_rn(Dn, X, bcast2(d4[1]));
                                Dn = __ffma2_rn(Dn, X, bcast2(d4[0]));
                                acc[m] = __ffma2_rn(__fmul2_rn(amp, N), make_float2(rcp_approx(Dn.x), rcp_approx(Dn.y)), acc[m]);
                            }
                            if (!__any_sync(0xffffffffu, member && !core)) continue;
                        }
                        const float2 c2 = bcast2((member && !core) ? rec.w : 0.f);
                        const bool far = all_far || (!none_far && (!member || core || o < fLr || o >= fRr));
                        if (all_far || (!none_far && __all_sync(0xffffffffu, far))) {
#pragma unroll
                            for (int m = 0; m < M; ++m) {
                                const float2 t = __fadd2_rn(xk[m], np2);
                                const float2 q = __ffma2_rn(t, t, g2);
                                if (m >= M - kNLDirect) {                          // (a share of the reciprocals taken one by one:
                                    acc[m] = __ffma2_rn(c2, make_float2(rcp_approx(q.x), rcp_approx(q.y)), acc[m]);   //  two instructions
                                    continue;                                      //  fewer, one more on the special-function unit)
                                }
                                const float R = rcp_approx(q.x * q.y);             // 1/q.x = R q.y, 1/q.y = R q.x
                                acc[m] = __ffma2_rn(c2, make_float2(R * q.y, R * q.x), acc[m]);
                            }
                        } else {
                            const float a2 = far ? 0.f : __int_as_float((int)((pk & 0x7FFFFu) << 12));
                            const float2 one = bcast2(1.0f), A1 = bcast2(1.5f * a2), nA2 = bcast2(-2.0f * a2 * rec.z);
#pragma unroll
                            for (int m = 0; m < M; ++m) {
                                const float2 t = __fadd2_rn(xk[m], np2);
                                const float2 q = __ffma2_rn(t, t, g2);
                                float2 rr;
                                if (m >= M - kNLDirect) rr = make_float2(rcp_approx(q.x), rcp_approx(q.y));
                                else { const float R = rcp_approx(q.x * q.y); rr = make_float2(R * q.y, R * q.x); }
                                const float2 uu = __ffma2_rn(nA2, rr, A1);
                                const float2 vv = __ffma2_rn(uu, rr, one);
                                const float2 ww = __fmul2_rn(rr, vv);
                                acc[m] = __ffma2_rn(c2, ww, acc[m]);
                            }
                        }
                    }
                };
                run(r.a0, r.a1); run(r.b0, r.b1); run(r.c0, r.c1); run(r.d0, r.d1);
                float v[kP];
#pragma unroll
                for (int m = 0; m < M; ++m) { v[2 * m] = acc[m].x; v[2 * m + 1] = acc[m].y; }
                warp_fold_add(a.node_acc + (size_t)sEnt[ei].e * kP, v, true, lane);
            }
            __syncthreads();                      // the entry list is rewritten by the next round
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) n_eval += __shfl_xor_sync(0xffffffffu, n_eval, o);
    if (lane == 0 && n_eval) atomicAdd(&a.st->pairs_node_eval, n_eval);
}

// Work is dealt in BLOCKS of kEdgeBlock consecutive sorted lines per warp (small enough for the second side to find the records in cache), one side at a time: along the sorted list the end
// bins are (nearly) non-decreasing, and in a dense list 32 consecutive lines end in the SAME bin for many batches in a
// row.  While that lasts the lanes just keep adding their node values in registers; the transposing fold and the 12
// atomics come once per run, when the warp-uniform bin changes (a batch whose lanes disagree goes through
// warp_add_by_bin as before).
constexpr int kEdgeBlock = 256;

__global__ void __launch_bounds__(kThreads, 3) edge_node_kernel(Params p, AccArgs a, const int32_t* __restrict__ keys,
                                                                 int32_t n)
{
    constexpr int M = kP / 2;
    __shared__ int32_t s_nact;
    apply_shift_bound(p, a.st);
    if (threadIdx.x == 0) s_nact = lower_bound_key(keys, n, (int64_t)p.ksent);
    __syncthreads();
    const int32_t n_act = s_nact;
    const int lane = threadIdx.x & 31;
    const int W = a.lv.w0;
    const int wshift = __ffs(a.lv.w0) - 1;
    float2 xk[M];
    const double hc = 0.5 * (double)(W - 1), hw = 0.5 * (double)W;
#pragma unroll
    for (int m = 0; m < M; ++m) xk[m] = make_float2((float)(hc + hw * kChebX[2 * m]), (float)(hc + hw * kChebX[2 * m + 1]));
    unsigned long long npairs = 0;
    const int warps_total = gridDim.x * (kThreads / 32), warp_global = blockIdx.x * (kThreads / 32) + (threadIdx.x >> 5);
    // (short lists: smaller blocks, so that every warp of the grid has one)
    const int blk_lines = 32 * max(1, min(kEdgeBlock / 32, n_act / (32 * warps_total)));
    const int n_blocks = (n_act + blk_lines - 1) / blk_lines;
    const float2 one = bcast2(1.0f);
    for (int blk = warp_global; blk < n_blocks; blk += warps_total) {
        const int i0 = blk * blk_lines, i1 = min(i0 + blk_lines, n_act);
#pragma unroll 1
        for (int side = 0; side < 2; ++side) {
            double* __restrict__ acc = a.edge_acc + (size_t)side * (size_t)a.N * kP;
            float run[kP];                        // this lane's share of the current run (all lanes: bin run_bin)
            int run_bin = -1;
            int key_T0 = -1;                      // the tile whose key threshold this lane computed last (fp64: kept)
            int64_t key_thr = 0;
#pragma unroll
            for (int j = 0; j < kP; ++j) run[j] = 0.f;
            // (the next batch's records are in flight while this one is evaluated)
            float4 rn_n = make_float4(0.f, 0.f, 1.f, 0.f), rb_n = make_float4(1.f, 0.f, __int_as_float(-1), 0.f);
            if (i0 + lane < i1) { rn_n = a.recN[i0 + lane]; rb_n = a.recB[i0 + lane]; }
#pragma unroll 1
            for (int ib = i0; ib < i1; ib += 32) {
                const int i = ib + lane;
                const bool live = i < i1;
                const float4 rn = rn_n, rb = rb_n;
                rn_n = make_float4(0.f, 0.f, 1.f, 0.f); rb_n = make_float4(1.f, 0.f, __int_as_float(-1), 0.f);
                if (i + 32 < i1) { rn_n = a.recN[i + 32]; rb_n = a.recB[i + 32]; }
                const int jc = __float_as_int(rn.x), ilo = __float_as_int(rb.y), ihi = __float_as_int(rb.z);
                const int e = side == 0 ? ihi : ilo;
                bool m = live && ihi >= ilo;
                const int T0 = m ? (e >> wshift) << wshift : 0;     // level-0 tiles are 64, 128 or 256 bins
                if (m) {
                    if (T0 != key_T0) { key_thr = side == 0 ? edge_key_upL(p, T0, W) : edge_key_dnR(p, T0, W); key_T0 = T0; }
                    m = side == 0 ? (int64_t)jc <= key_thr : (int64_t)jc >= key_thr;
                }
                // |z|^2 >= Z1 on the whole edge tile (the usual case: the extent ends many widths from the centre): one
                // asymptotic term; a line that needs two runs the same code with its a^2, so a warp takes one path and the
                // value of a pair never depends on its neighbours.  Every lane evaluates -- a lane without a pair with
                // amplitude 0 -- so that the batch runs without divergence
                const uint32_t pk = (uint32_t)__float_as_int(rn.y);
                const float a2 = __int_as_float((int)((pk & 0x7FFFFu) << 12));
                const float dist = (float)(side == 0 ? T0 - jc : jc - (T0 + W - 1)) - 1.0f;
                const bool far = !m || fmaf(dist, dist, rn.z) >= 1.001f * HK_Z1 * a2;
                const unsigned has = __ballot_sync(0xffffffffu, m);
                if (has == 0u) continue;
                npairs += m ? 1u : 0u;
                float v[kP];
                {
                    const float f = (float)(pk >> 19) * (1.0f / 8192.0f);
                    const float2 np2 = bcast2(-((float)(jc - T0) + f)), g2 = bcast2(rn.z), c2 = bcast2(m ? rn.w : 0.f);
                    if (__all_sync(0xffffffffu, far)) {
#pragma unroll
                        for (int mm = 0; mm < M; ++mm) {
                            const float2 t = __fadd2_rn(xk[mm], np2);
                            const float2 q = __ffma2_rn(t, t, g2);
                            float2 rr;                                       // (as node_lines_kernel: kNLDirect)
                            if (mm >= M - kNLDirect) rr = make_float2(rcp_approx(q.x), rcp_approx(q.y));
                            else { const float R = rcp_approx(q.x * q.y); rr = make_float2(R * q.y, R * q.x); }
                            const float2 ww = __fmul2_rn(c2, rr);
                            v[2 * mm] = ww.x; v[2 * mm + 1] = ww.y;
                        }
                    } else {
                        const float a2e = far ? 0.f : a2;
                        const float2 A1 = bcast2(1.5f * a2e), nA2 = bcast2(-2.0f * a2e * rn.z);
#pragma unroll
                        for (int mm = 0; mm < M; ++mm) {
                            const float2 t = __fadd2_rn(xk[mm], np2);
                            const float2 q = __ffma2_rn(t, t, g2);
                            float2 rr;
                            if (mm >= M - kNLDirect) rr = make_float2(rcp_approx(q.x), rcp_approx(q.y));
                            else { const float R = rcp_approx(q.x * q.y); rr = make_float2(R * q.y, R * q.x); }
                            const float2 uu = __ffma2_rn(nA2, rr, A1);
                            const float2 vv = __ffma2_rn(uu, rr, one);
                            const float2 ww = __fmul2_rn(c2, __fmul2_rn(rr, vv));
                            v[2 * mm] = ww.x; v[2 * mm + 1] = ww.y;
                        }
                    }
                }
                // the whole batch ends in the run's bin (lanes without a pair carry zeros): the common case
                if (run_bin >= 0 && __all_sync(0xffffffffu, !m || e == run_bin)) {
#pragma unroll
                    for (int j = 0; j < kP; ++j) run[j] += v[j];
                    continue;
                }
                // lanes that end in the run's bin join it; if the others agree on ONE bin (the list is sorted: a batch
                // straddles at most a bin boundary or two) the run is folded and a new one starts with them
                const bool in_run = m && e == run_bin;
                if (__any_sync(0xffffffffu, in_run)) {
#pragma unroll
                    for (int j = 0; j < kP; ++j) run[j] += in_run ? v[j] : 0.f;
                }
                const bool rest = m && !in_run;
                const unsigned rest_mask = __ballot_sync(0xffffffffu, rest);
                if (rest_mask == 0u) continue;
                if (run_bin >= 0) {                // the run ends here: fold it
                    warp_fold_add(acc + (size_t)run_bin * kP, run, true, lane);
                    run_bin = -1;
                }
                const int e1 = __shfl_sync(0xffffffffu, e, __ffs(rest_mask) - 1);
                if (__all_sync(0xffffffffu, !rest || e == e1)) {
                    run_bin = e1;
#pragma unroll
                    for (int j = 0; j < kP; ++j) run[j] = rest ? v[j] : 0.f;
                } else {
                    warp_add_by_bin(acc, rest ? (int64_t)e : -1, v, lane);
                }
            }
            if (run_bin >= 0) warp_fold_add(acc + (size_t)run_bin * kP, run, true, lane);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) npairs += __shfl_xor_sync(0xffffffffu, npairs, o);
    if (lane == 0 && npairs) atomicAdd(&a.st->pairs_edge_node, npairs);
}

// in place: side 0 -> suffix sums over each tile (bins <= the end bin), side 1 -> prefix sums (bins >= the start bin)
__global__ void __launch_bounds__(256) edge_scan_kernel(AccArgs a)
{
    const int64_t W = a.lv.w0;
    const int64_t n_tiles = (a.N + W - 1) / W;
    const int64_t idx = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (idx >= 2 * n_tiles * kP) return;
    const int j = (int)(idx % kP);
    const int64_t tile = (idx / kP) % n_tiles;
    const int side = (int)(idx / (kP * n_tiles));
    double* __restrict__ acc = a.edge_acc + (size_t)side * (size_t)a.N * kP;
    const int64_t b0 = tile * W, b1 = min(a.N, b0 + W);
    double run = 0.0;
    if (side == 0) {
        for (int64_t b = b1 - 1; b >= b0; --b) { run += acc[(size_t)b * kP + j]; acc[(size_t)b * kP + j] = run; }
    } else {
        for (int64_t b = b0; b < b1; ++b) { run += acc[(size_t)b * kP + j]; acc[(size_t)b * kP + j] = run; }
    }
}

// value at xi (tile-normalised coordinate in [-1, 1]) of the degree-(kP-1) interpolant through the node sums
__device__ __forceinline__ double cheb_interp(const double* __restrict__ nodes, double xi)
{
    double num = 0.0, den = 0.0;
#pragma unroll
    for (int k = 0; k < kP; ++k) {
        const double d = xi - kChebX[k];
        if (d == 0.0) return nodes[k];
        const double w = kChebW[k] / d;
        num = fma(w, nodes[k], num);
        den += w;
    }
    return num / den;
}

// level l -> l - 1: restriction of the parent's polynomial to each child's nodes (exact for polynomials)
__global__ void __launch_bounds__(256) node_down_kernel(AccArgs a, int l)
{
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    const int n_child = a.lv.off[l] - a.lv.off[l - 1];
    if (idx >= n_child * kP) return;
    const int jc = idx / kP, kk = idx - jc * kP;
    const double xi = ((jc & 1) ? 0.5 : -0.5) + 0.5 * kChebX[kk];
    const double v = cheb_interp(a.node_acc + (size_t)(a.lv.off[l] + (jc >> 1)) * kP, xi);
    if (v != 0.0) a.node_acc[(size_t)(a.lv.off[l - 1] + jc) * kP + kk] += v;
}

// level-0 node sums -> bins of k(nu)
__global__ void __launch_bounds__(256) node_bins_kernel(AccArgs a)
{
    const int64_t b = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (b >= a.N) return;
    const int64_t j = b / a.lv.w0;
    const double xi = ((double)(b - j * a.lv.w0) - 0.5 * (double)(a.lv.w0 - 1)) / (0.5 * (double)a.lv.w0);
    const double v = cheb_interp(a.node_acc + (size_t)j * kP, xi);
    if (v != 0.0) a.out_k[b] += v * scalbn(1.0, -a.st->scale_exp);
}

// scanned edge accumulators -> bins of k(nu)
__global__ void __launch_bounds__(256) edge_bins_kernel(AccArgs a)
{
    const int64_t b = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (b >= a.N) return;
    const double* __restrict__ r0 = a.edge_acc + (size_t)b * kP;
    const double* __restrict__ r1 = a.edge_acc + ((size_t)a.N + (size_t)b) * kP;
    double nodes[kP];
    bool any = false;
#pragma unroll
    for (int j = 0; j < kP; ++j) { nodes[j] = r0[j] + r1[j]; any |= nodes[j] != 0.0; }
    if (!any) return;
    const int64_t j0 = b / a.lv.w0;
    const double xi = ((double)(b - j0 * a.lv.w0) - 0.5 * (double)(a.lv.w0 - 1)) / (0.5 * (double)a.lv.w0);
    a.out_k[b] += cheb_interp(nodes, xi) * scalbn(1.0, -a.st->scale_exp);
}

// ---------------------------------------------------------------------------------------
// plinth removal (section 2.1.1): subtract S V(cut) of every line from every bin of its extent
// ---------------------------------------------------------------------------------------
// The removed part is a sum of boxes, one per line: -p_l on [ilo, ihi].  Lanes walk the lines, evaluate p_l from the
// SAME fp32 widths the accumulation kernels use (so V - V(cut) goes to zero consistently at the extent's ends) with
// the same region split, and add -p_l at ilo and +p_l at ihi + 1 of a difference array (equal bins summed
// in the warp first); a running sum over the bins (CUB) turns it into the box sum, plinth_apply_kernel adds it to k.
__device__ __forceinline__ void warp_add_scalar_by_bin(double* __restrict__ acc, int64_t bin, double v, int lane)
{
    unsigned todo = __ballot_sync(0xffffffffu, bin >= 0);
    while (todo) {
        const int leader = __ffs(todo) - 1;
        const int64_t b = __shfl_sync(0xffffffffu, bin, leader);
        const bool mine = (bin == b);
        const unsigned grp = __ballot_sync(0xffffffffu, mine);
        double sum = mine ? v : 0.0;
        if (__popc(grp) > 1) {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
        }
        if (lane == leader) atomicAdd(acc + b, sum);
        todo &= ~grp;
    }
}

__global__ void __launch_bounds__(256) plinth_kernel(Params p, AccArgs a, const RecU* __restrict__ rec, int64_t n)
{
    // over the UNSORTED per-line records: they hold the true widths (the profile variants zero one of them only in the
    // sorted records), which a width-relative cutting length needs, and the unscaled fp64 amplitude
    const int lane = threadIdx.x & 31;
    const int64_t n_round = (n + 31) & ~31LL;
    unsigned long long in_core = 0;        // lines whose value at the cut is not small against their peak (hk_stats.n_plinth_illcond)
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n_round; i += (int64_t)gridDim.x * blockDim.x) {
        int64_t ilo = 0, ihi = -1;
        double pl = 0.0;
        if (i < n) {
            const RecU r = rec[i];
            ilo = r.ilo; ihi = r.ihi;
            if (ihi >= ilo) {
                const double G2t = (double)r.G2, a2 = (double)r.a2;
                // the line's own cutting length in bins
                const double cb = p.cut_mode == 0 ? p.cut_bins
                                : p.cut_factor * (p.cut_mode == 1 ? sqrt(G2t) : sqrt(a2) * 0.83255461115769775635);
                const bool gauss = p.profile == HK_PROFILE_DOPPLER || p.profile == HK_PROFILE_BINNED_GAUSSIAN;
                const double G2 = gauss ? 0.0 : G2t;
                const double q = cb * cb + G2;
                const double c = r.cK * sqrt(G2 * a2) * 0.56418958354775628695;        // Lorentz amplitude, as gather_kernel
                double peak = 0.0;                                                      // the line's value at its centre
                if (p.profile == HK_PROFILE_BINNED_GAUSSIAN) {
                    if (q < (double)binned_ql(r.a2)) pl = r.cK * (double)binned_K((float)cb, 0.f, 0.f, rsqrtf(r.a2));
                    peak = r.cK * (double)binned_K(0.f, 0.f, 0.f, rsqrtf(r.a2));
                } else if (p.profile == HK_PROFILE_LORENTZ) {
                    pl = c / q;
                    peak = c / G2;
                } else {
                    // two asymptotic terms in bin units: c/q (1 + (1.5 a^2 - 2 a^2 G^2/q)/q); inside the core the fp32 evaluator
                    const float inv_a = rsqrtf(r.a2);
                    const float y = sqrtf((float)G2) * inv_a;
                    if (q >= (double)HK_Z2 * a2) pl = c / q * (1.0 + (1.5 * a2 - 2.0 * a2 * G2 / q) / q);
                    else {
                        const float x = (float)cb * inv_a;
                        // (a pure Gaussian through the same scaled fp32 evaluation as its bins, so that both vanish together)
                        pl = y == 0.f ? (double)gauss_term((float)scalbn(r.cK, a.st->scale_exp), x) * scalbn(1.0, -a.st->scale_exp)
                                      : r.cK * (double)core_any_K(x, y, nullptr);
                    }
                    peak = G2 >= (double)HK_Z2 * a2 ? c / G2 * (1.0 - 0.5 * a2 / G2) : y == 0.f ? r.cK : r.cK * (double)core_any_K(0.f, y, nullptr);
                }
                // S (V - V(cut)) is ill-conditioned in fp32 when V(cut) is not small against the peak (hk.h, hk_set_plinth)
                if (pl * (double)HK_PLINTH_RATIO > peak) ++in_core;
            }
        }
        const bool live = ihi >= ilo;
        warp_add_scalar_by_bin(a.plinth_acc, live ? ilo : -1, -pl, lane);
        warp_add_scalar_by_bin(a.plinth_acc, live ? ihi + 1 : -1, pl, lane);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) in_core += __shfl_xor_sync(0xffffffffu, in_core, o);
    if (lane == 0 && in_core) atomicAdd(&a.st->n_plinth_illcond, in_core);
}

__global__ void __launch_bounds__(256) plinth_apply_kernel(AccArgs a)
{
    const int64_t b = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (b >= a.N) return;
    const double v = a.plinth_acc[b];              // running sum: minus the plinths of the lines that cover bin b
    if (v != 0.0) a.out_k[b] += v;
}

// ---------------------------------------------------------------------------------------
// accuracy probe: the same device functions on a lattice of (x, y), alpha_D = 1 bin
// ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) probe_kernel(const float* __restrict__ x, const float* __restrict__ y, int64_t n,
                                                    float* __restrict__ out, int32_t* __restrict__ region)
{
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const float t = x[i], G = y[i];
        const float G2 = G * G, q = fmaf(t, t, G2);
        const float c = G * 0.564189583547756f;          // Lorentz amplitude of Re w: y/sqrt(pi)
        float K;
        int reg;
        if (q >= HK_Z1) { K = term_far(c, q); reg = 0; }
        else if (q >= HK_Z2) { K = c * shape_mid(rcp_approx(q), 1.5f, 2.0f * G2); reg = 1; }
        else {
            K = core_any_K(fabsf(t), G, &reg);
            // regions 2 and 3 as the row kernel evaluates them: the expanded rational forms (hk_centre.cuh)
            if (reg == 2) K = gh4_row_K(t * t, G2, G);
            if (reg == 3) K = gh6_row_K(t * t, G2, G);
            if (reg == 5) K = gh10_row_K(t * t, G2, G);
        }
        out[i] = K;
        if (region) region[i] = reg;
    }
}

// ---------------------------------------------------------------------------------------
// FP32 issue-rate probes (roofline denominator): 16 independent register-resident chains per thread.
// kind 0: FFMA2 with three distinct register operands   1: scalar FFMA, three register operands
//      2: FFMA2 whose multiplier and addend are scalars broadcast to both halves (the row kernels' form)
//      3: FADD2   4: FMUL2   5: MUFU.RCP (one per chain step)
// clk[0] = SM cycles (clock64) and clk[1] = nanoseconds (globaltimer) block 0 spent in the loop: their ratio is the SM
// clock actually held while the probe ran.
// ---------------------------------------------------------------------------------------
template <int kKind>
__global__ void __launch_bounds__(512) fp32_probe_kernel(int iters, float* __restrict__ sink, long long* __restrict__ clk)
{
    float2 acc[16];
#pragma unroll
    for (int j = 0; j < 16; ++j) acc[j] = make_float2(1.0f + j + threadIdx.x * 1e-3f, 0.5f + j);
    const float2 a = make_float2(0.999999f, 1.000001f), b = make_float2(1e-7f, -1e-7f);
    const long long t0 = clock64();
    unsigned long long g0, g1;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g0));
#pragma unroll 1
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            if (kKind == 0) acc[j] = __ffma2_rn(acc[j], a, b);
            else if (kKind == 1) { acc[j].x = fmaf(acc[j].x, a.x, b.x); acc[j].y = fmaf(acc[j].y, a.y, b.y); }
            else if (kKind == 2) acc[j] = __ffma2_rn(acc[j], make_float2(a.x, a.x), make_float2(b.x, b.x));
            else if (kKind == 3) acc[j] = __fadd2_rn(acc[j], b);
            else if (kKind == 4) acc[j] = __fmul2_rn(acc[j], a);
            else acc[j].x = rcp_approx(acc[j].x);
        }
    }
    const long long t1 = clock64();
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g1));
    float s = 0.f;
#pragma unroll
    for (int j = 0; j < 16; ++j) s += acc[j].x + acc[j].y;
    if (s == 123.456f) *sink = s;
    if (threadIdx.x == 0 && blockIdx.x == 0) { clk[0] = t1 - t0; clk[1] = (long long)(g1 - g0); }
}

}  // namespace hk
