// hk_accumulate.cuh -- steps a4-a7 of the hot path: the two accumulation
// kernels.  Both are output-stationary: a CTA owns kTileBins consecutive bins, a warp owns
// kWarpBins of them, a lane owns kB bins (lane + 32 j) in registers.  Lines arrive sorted by
// centre bin, so the lines that can reach a tile are one contiguous index range; a work unit
// is (CTA tile, chunk of that range) and units are handed out by an atomic counter to a
// persistent grid (one wave, multiples of the SM count).  fp32 partial sums are flushed into
// fp64 registers every kFlush lines and reach k(nu) with one fp64 atomic per bin per unit.
//
//   far_kernel  : pairs whose whole warp tile is inside the extent and has |z|^2 >= Z1:
//                 branch-free Lorentzian, two lines share one reciprocal, packed fp32 (FFMA2).
//   near_kernel : everything else (extent edges, |z|^2 < Z1): exact integer extent mask,
//                 two-term asymptotic, and the core evaluator where |z|^2 < Z2.
//
// The paper's kernel (L243-330) walks lines in threads and nu-points serially with a
// shared-memory K_s and four launches per block (AL/AR/B/C, L354); what is kept is the idea
// of formula-uniform launches.
#pragma once
#include "hk_preprocess.cuh"

namespace hk {

struct AccArgs {
    const float4* __restrict__ recA;
    const float4* __restrict__ recB;
    const TileRange* __restrict__ tr;
    const int32_t* __restrict__ unit_prefix;   // n_ct + 1 entries (exclusive scan of counts)
    DevStats* st;
    double* __restrict__ out_k;
    int64_t N;
    int32_t n_wt, n_ct, chunk;
};

// Which CTA tile does unit u belong to?  Largest ct with prefix[ct] <= u.
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

// ---------------------------------------------------------------------------------------
// far kernel
// ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kThreads, 2) far_kernel(AccArgs a)
{
    __shared__ float4 sm[kSub];       // { -tl, G2, c, - } with tl = centre position relative to the CTA tile
    __shared__ int s_unit;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int total = a.unit_prefix[a.n_ct];

    float2 tb[kB / 2];
#pragma unroll
    for (int m = 0; m < kB / 2; ++m) {
        float b0 = (float)(warp * kWarpBins + lane + 64 * m);
        tb[m] = make_float2(b0, b0 + 32.0f);
    }

    for (;;) {
        const int u = next_unit(&a.st->unit_counter_far, &s_unit);
        if (u >= total) break;
        const int ct = find_tile(a.unit_prefix, a.n_ct, u);
        const int wt_first = ct * kWarps, wt_last = min(a.n_wt, wt_first + kWarps) - 1;
        const int64_t ct0 = (int64_t)ct * kTileBins;
        const int cA0 = a.tr[wt_first].A0, cA1 = a.tr[wt_last].A1;
        const int c0 = cA0 + (u - a.unit_prefix[ct]) * a.chunk;
        const int c1 = min(c0 + a.chunk, cA1);
        const int wt = wt_first + warp;
        int fl0 = 0, fl1 = 0, fr0 = 0, fr1 = 0;
        if (wt <= wt_last) {
            TileRange r = a.tr[wt];
            fl0 = max(r.FL0, c0); fl1 = min(r.FL1, c1);
            fr0 = max(r.FR0, c0); fr1 = min(r.FR1, c1);
        }
        if (!__syncthreads_or((fl0 < fl1) || (fr0 < fr1))) continue;
        if (threadIdx.x == 0) atomicAdd(&a.st->units_far, 1ULL);

        float2 acc[kB / 2];
        double acc64[kB];
#pragma unroll
        for (int m = 0; m < kB / 2; ++m) acc[m] = make_float2(0.f, 0.f);
#pragma unroll
        for (int j = 0; j < kB; ++j) acc64[j] = 0.0;
        int since_flush = 0;

        for (int s0 = c0; s0 < c1; s0 += kSub) {
            const int s1 = min(s0 + kSub, c1);
            const int p0 = max(fl0, s0), p1 = min(fl1, s1);
            const int q0 = max(fr0, s0), q1 = min(fr1, s1);
            if (!__syncthreads_or((p0 < p1) || (q0 < q1))) continue;   // also fences reuse of sm
            for (int i = threadIdx.x; i < s1 - s0; i += kThreads) {
                float4 r = a.recA[s0 + i];
                float tl = (float)((int64_t)__float_as_int(r.x) - ct0) + r.y;
                sm[i] = make_float4(-tl, r.z, r.w, 0.f);
            }
            __syncthreads();
#pragma unroll 1
            for (int seg = 0; seg < 2; ++seg) {
                int l = (seg == 0 ? p0 : q0) - s0;
                const int le = (seg == 0 ? p1 : q1) - s0;
                while (l < le) {
                    const int stop = min(le, l + (kFlush - since_flush));
                    since_flush += stop - l;
                    for (; l + 1 < stop; l += 2) {
                        const float4 r1 = sm[l], r2 = sm[l + 1];
                        const float2 n1 = make_float2(r1.x, r1.x), g1 = make_float2(r1.y, r1.y), c1 = make_float2(r1.z, r1.z);
                        const float2 n2 = make_float2(r2.x, r2.x), g2 = make_float2(r2.y, r2.y), c2 = make_float2(r2.z, r2.z);
#pragma unroll
                        for (int m = 0; m < kB / 2; ++m) {
                            // c1/q1 + c2/q2 = (c1 q2 + c2 q1) / (q1 q2): one reciprocal for two lines
                            float2 t1 = __fadd2_rn(tb[m], n1);
                            float2 t2 = __fadd2_rn(tb[m], n2);
                            float2 q1 = __ffma2_rn(t1, t1, g1);
                            float2 q2 = __ffma2_rn(t2, t2, g2);
                            float2 pp = __fmul2_rn(q1, q2);
                            float2 nn = __fmul2_rn(c1, q2);
                            nn = __ffma2_rn(c2, q1, nn);
                            float2 rr = make_float2(rcp_approx(pp.x), rcp_approx(pp.y));
                            acc[m] = __ffma2_rn(nn, rr, acc[m]);
                        }
                    }
                    if (l < stop) {       // odd line out
                        const float4 r1 = sm[l];
                        const float2 n1 = make_float2(r1.x, r1.x), g1 = make_float2(r1.y, r1.y), c1 = make_float2(r1.z, r1.z);
#pragma unroll
                        for (int m = 0; m < kB / 2; ++m) {
                            float2 t1 = __fadd2_rn(tb[m], n1);
                            float2 q1 = __ffma2_rn(t1, t1, g1);
                            float2 rr = make_float2(rcp_approx(q1.x), rcp_approx(q1.y));
                            acc[m] = __ffma2_rn(c1, rr, acc[m]);
                        }
                        ++l;
                    }
                    if (since_flush >= kFlush) {
#pragma unroll
                        for (int m = 0; m < kB / 2; ++m) {
                            acc64[2 * m] += (double)acc[m].x;
                            acc64[2 * m + 1] += (double)acc[m].y;
                            acc[m] = make_float2(0.f, 0.f);
                        }
                        since_flush = 0;
                    }
                }
            }
        }
        const double inv_scale = scalbn(1.0, -a.st->scale_exp);
#pragma unroll
        for (int m = 0; m < kB / 2; ++m) {
            const int64_t b = ct0 + warp * kWarpBins + lane + 64 * m;
            double v0 = (acc64[2 * m] + (double)acc[m].x) * inv_scale;
            double v1 = (acc64[2 * m + 1] + (double)acc[m].y) * inv_scale;
            if (b < a.N && v0 != 0.0) atomicAdd(a.out_k + b, v0);
            if (b + 32 < a.N && v1 != 0.0) atomicAdd(a.out_k + b + 32, v1);
        }
    }
}

// ---------------------------------------------------------------------------------------
// near / edge kernel
// ---------------------------------------------------------------------------------------
template <bool kCore>
__device__ __forceinline__ void near_line(const float4 ra, const float4 rb, const float (&tb)[kB], float (&acc)[kB])
{
    const float dlt = ra.x, f = ra.y, G2 = ra.z, c = ra.w;
    const float a2 = rb.x, lo = rb.y, hi = rb.z, cK = rb.w;
    const float A1 = 1.5f * a2, A2 = 2.0f * a2 * G2;
    const float qc = HK_Z2 * a2;
    float inv_a = 0.f, y = 0.f;
    if (kCore) {
        inv_a = rsqrtf(a2);
        y = sqrtf(G2) * inv_a;
    }
#pragma unroll
    for (int j = 0; j < kB; ++j) {
        const float d = tb[j] - dlt;            // exact: both are small integers
        const float t = d - f;
        const float q = fmaf(t, t, G2);
        const bool in = (tb[j] >= lo) && (tb[j] <= hi);       // exact integer extent (R7)
        const float r = rcp_approx(q);
        const float term = c * shape_mid(r, A1, A2);
        if (kCore) {
            const bool core = in && (q < qc);
            if (in && !core) acc[j] += term;
            if (__any_sync(0xffffffffu, core)) {
                if (core) acc[j] = fmaf(cK, core_K(fabsf(t) * inv_a, y), acc[j]);
            }
        } else {
            if (in) acc[j] += term;
        }
    }
}

__global__ void __launch_bounds__(kThreads, 2) near_kernel(AccArgs a)
{
    __shared__ float4 smA[kSub];   // { jc - ct0, f, G2, c }
    __shared__ float4 smB[kSub];   // { a2, ilo - ct0, ihi - ct0, cK }   (as floats, exact integers)
    __shared__ int s_unit;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int total = a.unit_prefix[a.n_ct];
    const float wlo = (float)(warp * kWarpBins), whi = wlo + (float)(kWarpBins - 1);

    float tb[kB];
#pragma unroll
    for (int j = 0; j < kB; ++j) tb[j] = (float)(warp * kWarpBins + lane + 32 * j);

    for (;;) {
        const int u = next_unit(&a.st->unit_counter_near, &s_unit);
        if (u >= total) break;
        const int ct = find_tile(a.unit_prefix, a.n_ct, u);
        const int wt_first = ct * kWarps, wt_last = min(a.n_wt, wt_first + kWarps) - 1;
        const int64_t ct0 = (int64_t)ct * kTileBins;
        const int cA0 = a.tr[wt_first].A0, cA1 = a.tr[wt_last].A1;
        const int c0 = cA0 + (u - a.unit_prefix[ct]) * a.chunk;
        const int c1 = min(c0 + a.chunk, cA1);
        const int wt = wt_first + warp;
        int g0[3] = {0, 0, 0}, g1[3] = {0, 0, 0};
        if (wt <= wt_last) {
            TileRange r = a.tr[wt];
            g0[0] = max(r.A0, c0);  g1[0] = min(r.FL0, c1);
            g0[1] = max(r.FL1, c0); g1[1] = min(r.FR0, c1);
            g0[2] = max(r.FR1, c0); g1[2] = min(r.A1, c1);
        }
        if (!__syncthreads_or((g0[0] < g1[0]) || (g0[1] < g1[1]) || (g0[2] < g1[2]))) continue;
        if (threadIdx.x == 0) atomicAdd(&a.st->units_near, 1ULL);

        float acc[kB];
        double acc64[kB];
#pragma unroll
        for (int j = 0; j < kB; ++j) { acc[j] = 0.f; acc64[j] = 0.0; }
        int since_flush = 0;

        for (int s0 = c0; s0 < c1; s0 += kSub) {
            const int s1 = min(s0 + kSub, c1);
            int p0[3], p1[3];
            bool mine = false;
#pragma unroll
            for (int s = 0; s < 3; ++s) {
                p0[s] = max(g0[s], s0); p1[s] = min(g1[s], s1);
                mine |= p0[s] < p1[s];
            }
            if (!__syncthreads_or(mine)) continue;
            for (int i = threadIdx.x; i < s1 - s0; i += kThreads) {
                float4 ra = a.recA[s0 + i], rb = a.recB[s0 + i];
                const int64_t lim = 1 << 24;
                int64_t dj = (int64_t)__float_as_int(ra.x) - ct0;
                int64_t dlo = (int64_t)__float_as_int(rb.y) - ct0, dhi = (int64_t)__float_as_int(rb.z) - ct0;
                dlo = max(-lim, min(lim, dlo));
                dhi = max(-lim, min(lim, dhi));
                smA[i] = make_float4((float)dj, ra.y, ra.z, ra.w);
                smB[i] = make_float4(rb.x, (float)dlo, (float)dhi, rb.w);
            }
            __syncthreads();
#pragma unroll 1
            for (int s = 0; s < 3; ++s) {
#pragma unroll 1
                for (int l = p0[s] - s0; l < p1[s] - s0; ++l) {
                    const float4 ra = smA[l], rb = smB[l];
                    // can |z|^2 < Z2 occur anywhere in this warp's bins?  (warp-uniform)
                    const float pos = ra.x + ra.y;
                    const float dist = fmaxf(0.f, fmaxf(wlo - pos, pos - whi));
                    if (fmaf(dist, dist, ra.z) < HK_Z2 * rb.x) near_line<true>(ra, rb, tb, acc);
                    else near_line<false>(ra, rb, tb, acc);
                    if (++since_flush >= kFlush) {
#pragma unroll
                        for (int j = 0; j < kB; ++j) { acc64[j] += (double)acc[j]; acc[j] = 0.f; }
                        since_flush = 0;
                    }
                }
            }
        }
        const double inv_scale = scalbn(1.0, -a.st->scale_exp);
#pragma unroll
        for (int j = 0; j < kB; ++j) {
            const int64_t b = ct0 + warp * kWarpBins + lane + 32 * j;
            double v = (acc64[j] + (double)acc[j]) * inv_scale;
            if (b < a.N && v != 0.0) atomicAdd(a.out_k + b, v);
        }
    }
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
        else { K = core_K(fabsf(t), G); reg = 2; }
        out[i] = K;
        if (region) region[i] = reg;
    }
}

// ---------------------------------------------------------------------------------------
// FP32 issue-rate probe (roofline denominator): 32 independent FMA chains per thread
// ---------------------------------------------------------------------------------------
template <bool kPacked>
__global__ void __launch_bounds__(512) fp32_peak_kernel(int iters, float* __restrict__ sink)
{
    float2 acc[16];
#pragma unroll
    for (int j = 0; j < 16; ++j) acc[j] = make_float2(1.0f + j + threadIdx.x * 1e-3f, 0.5f + j);
    const float2 a = make_float2(0.999999f, 1.000001f), b = make_float2(1e-7f, -1e-7f);
#pragma unroll 1
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            if (kPacked) acc[j] = __ffma2_rn(acc[j], a, b);
            else { acc[j].x = fmaf(acc[j].x, a.x, b.x); acc[j].y = fmaf(acc[j].y, a.y, b.y); }
        }
    }
    float s = 0.f;
#pragma unroll
    for (int j = 0; j < 16; ++j) s += acc[j].x + acc[j].y;
    if (s == 123.456f) *sink = s;
}

}  // namespace hk
