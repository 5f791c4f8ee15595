// matched_filter_warp.cu -- baseline removal by running mean + boxcar matched filters: the warp-autonomous kernel
// used for the passes that store no dense z (RMS + block maxima only; sparse re-computation of single blocks) --
// dedisp_search_events and dedisp_matched_filter_rms(z_dev = NULL).  matched_filter.cu holds the CTA-cooperative
// kernel that writes the dense z.
// (Sec. 2.3), one streaming pass over
// the dedispersed time series, HBM-bound.
//
//   y[t]   = x[t] - (1/N) sum_{k=a(t)}^{a(t)+N-1} x[k],  N = 2R+1, a(t) = clip(t-R, 0, n-N)
//   z_w[t] = (1/sqrt(w)) sum_{k<w} y[t+k]   for t <= n-w,   0 beyond
//
// The paper's algorithm is "prefix sum, then subtract the points at plus and minus
// the window radius", and the same again for the boxcars.  Here both prefix sums are
// carried along a row segment in exact modular integers:
//   Wsum[t] = Wsum[t-1] + (x[t+R] - x[t-R-1])           (running window sum, scan of d)
//   NY[t]   = N*x[t] - Wsum[t]                           (N * baseline-removed sample)
//   P[t+1]  = P[t] + NY[t]                               (prefix sum of NY, kept in a ring)
//   z_w[t]  = float(P[t+w] - P[t]) * fl32(1 / (N sqrt(w)))
// Differences of modular prefix sums are exact as long as the true value fits the
// word, so 32-bit words serve whenever wmax*N*x_max < 2^31 (or, guarded by a per-step
// check of the data, whenever N*x_max < 2^31) and 64-bit words otherwise.
//
// Round-2 design: WARP-AUTONOMOUS.  A work item is (row, segment of SEG samples) and belongs to ONE warp, which
// walks it in steps of 32 x 8 = 256 samples with nothing but warp shuffles and its own shared-memory ring: no
// __syncthreads() anywhere.  Round 1 gave a segment to a 256-thread CTA (2048-sample steps, two block scans and
// seven barriers per step): ncu showed 892 warp instructions per step and warp, issue slots 54 % busy, the rest
// barrier and scoreboard stalls (profiles/r2_matched_filter.md).  Per step a lane
//   * loads its 8 consecutive samples of x, x[t+R] and x[t-R-1] with 128-bit loads straight into registers (the two
//     shifted streams as three aligned vectors + a register pick; scalar loads at row ends and for unaligned rows),
//   * scans d and NY across the warp with shuffles, appends 8 prefix sums to the ring (two 128-bit stores),
//   * emits 8 outputs per width that lag L (wmax rounded up to 4) samples behind, four at a time: 128-bit ring
//     reads (two vectors + a pick when the width is not a multiple of 4), one 128-bit streaming store per four
//     outputs (scalar path: row ends, unaligned rows, 64-bit words, the guard's slow steps).
#include <cmath>
#include <type_traits>

#include "dedisp_internal.h"

// resident warps per SM the register budget is set for: CTAs of 2 warps, MF_MINB of them per SM
#ifndef MF_MINB
#define MF_MINB 18
#endif

namespace {

constexpr int V = 8;             // samples per lane per step
constexpr int WS = 32 * V;       // samples per warp step
constexpr int WPB = 2;           // (independent) warps per CTA
constexpr int NT = 32 * WPB;
constexpr int E = 2048;          // outputs per block of the block-maximum hint (dedisp_find_events_hinted)
constexpr int MAXW = 16;         // boxcar widths per call
constexpr int PB = 256;          // samples per block of the per-row prefix sums
static_assert(E % WS == 0, "a hint block is a whole number of warp steps");

struct MFParams {
    const void *x;               // [nrows][n] uint32 or float32 (exact integers)
    float *z;                    // [nw][nrows][n], or null (RMS / block maxima only)
    long long nrows, n;
    long long nitems;            // dense: work items of this launch = rows of the launch * nseg
    long long row0;              // dense: first row of this launch (rows are processed in L2-sized blocks)
    long long plane;             // elements between the outputs of consecutive widths (nrows * n; 0 in sparse mode)
    int radius;
    int nw;
    int wmax;
    int lag;                     // wmax rounded up to a multiple of 4: outputs trail the inputs of a step by this much
    int vec_in, vec_out;         // x rows / z rows are 16-byte aligned (base pointer and n multiple of 4 words)
    int ring;                    // ring entries per warp, multiple of 8, >= WS + lag + 8
    int warp_smem;               // shared-memory bytes per warp
    int seg;                     // samples per segment (multiple of E)
    int nseg;
    int guard_lim;               // guarded 32-bit mode: |NY| <= guard_lim => every boxcar fits int32
    unsigned long long guard_hist;   // mask of the step flags the outputs of one step depend on
    int w[MAXW];
    int wl[MAXW];                // width indices: those with w % 4 == 0 first (n4 of them), then the others
    int n4;
    float scale[MAXW];           // fl32(1 / (N sqrt(w)))
    double *partial;             // RMS variant: [nw][nrows][nseg] sums of z^2 over a segment
    int *blockmax;               // RMS variant, optional: [nw][nrows][nblk] upper bounds of z per block of E outputs
    int nblk;
    // sparse re-computation (dedisp_search_events): warp i re-runs the steps that produce block sparse_list[i].y of
    // series sparse_list[i].x (= width index * nrows + row) and stores that block's E outputs at zc + i*E
    // per-row prefix sums of x at multiples of PB samples (mf_prefix_kernel): prefix[row * (pnb + 1) + k] =
    // sum of x[row][0 .. min(k * PB, n)); the window sum at the start of a work item is then two look-ups and two
    // edges of < PB samples instead of a sum over N = 2R + 1 samples -- which makes short segments affordable
    const unsigned long long *prefix;
    int pnb;
    const int2 *sparse_list;     // nullptr: the dense pass
    const int *sparse_count;     // number of valid entries (device)
    float *zc;
};

// inclusive warp scan; returns the lane's inclusive prefix and the warp total
template <class ACC>
__device__ __forceinline__ ACC warp_scan(ACC v, ACC &total)
{
    const int lane = threadIdx.x & 31;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const ACC u = __shfl_up_sync(0xffffffffu, v, o);
        if (lane >= o) v += u;
    }
    total = __shfl_sync(0xffffffffu, v, 31);
    return v;
}

template <bool XF32>
__device__ __forceinline__ uint32_t cvt_x(uint32_t raw)
{
    return XF32 ? (uint32_t)__uint_as_float(raw) : raw;
}

// float32 of a signed accumulator; the 64-bit conversion runs on the slow XU pipe, so
// numerators that fit 32 bits (almost all) take the fast conversion -- same rounding.
__device__ __forceinline__ float acc_to_float(uint32_t d) { return (float)(int)d; }
__device__ __forceinline__ float acc_to_float(unsigned long long d)
{
    const int l = (int)(uint32_t)d, h = (int)(uint32_t)(d >> 32);
    if (h == (l >> 31)) return (float)l;
    return (float)(long long)d;
}

template <class ACC> struct Vec8;
template <> struct Vec8<uint32_t> {
    static __device__ __forceinline__ void store(uint32_t *p, const uint32_t (&v)[V])
    {
        reinterpret_cast<uint4 *>(p)[0] = make_uint4(v[0], v[1], v[2], v[3]);
        reinterpret_cast<uint4 *>(p)[1] = make_uint4(v[4], v[5], v[6], v[7]);
    }
};
template <> struct Vec8<unsigned long long> {
    static __device__ __forceinline__ void store(unsigned long long *p, const unsigned long long (&v)[V])
    {
#pragma unroll
        for (int q = 0; q < 4; ++q)
            reinterpret_cast<ulonglong2 *>(p)[q] = make_ulonglong2(v[2 * q], v[2 * q + 1]);
    }
};

// words a .. a+7 of the 12 words held by three aligned 16-byte vectors (a = 0..3, warp-uniform)
__device__ __forceinline__ void pick8(const uint4 &v0, const uint4 &v1, const uint4 &v2, int a, uint32_t (&o)[8])
{
    const uint32_t w[12] = {v0.x, v0.y, v0.z, v0.w, v1.x, v1.y, v1.z, v1.w, v2.x, v2.y, v2.z, v2.w};
    if (a == 0) {
#pragma unroll
        for (int k = 0; k < 8; ++k) o[k] = w[k];
    } else if (a == 1) {
#pragma unroll
        for (int k = 0; k < 8; ++k) o[k] = w[k + 1];
    } else if (a == 2) {
#pragma unroll
        for (int k = 0; k < 8; ++k) o[k] = w[k + 2];
    } else {
#pragma unroll
        for (int k = 0; k < 8; ++k) o[k] = w[k + 3];
    }
}
// words a .. a+3 of the 8 words of two vectors
__device__ __forceinline__ void pick4(const uint4 &v0, const uint4 &v1, int a, uint32_t (&o)[4])
{
    if (a == 0) { o[0] = v0.x; o[1] = v0.y; o[2] = v0.z; o[3] = v0.w; }
    else if (a == 1) { o[0] = v0.y; o[1] = v0.z; o[2] = v0.w; o[3] = v1.x; }
    else if (a == 2) { o[0] = v0.z; o[1] = v0.w; o[2] = v1.x; o[3] = v1.y; }
    else { o[0] = v0.w; o[1] = v1.x; o[2] = v1.y; o[3] = v1.z; }
}

__device__ __forceinline__ int ordered_int(float v)
{
    const int o = __float_as_int(v);
    return o >= 0 ? o : o ^ 0x7fffffff;
}

// GUARD (32-bit words only, host has checked N*x_max < 2^31 so that NY is exact in int32):
// the worst-case boxcar wmax*N*x_max does not fit 32 bits, but real series stay far below
// it.  Every step flags |NY| > (2^31-1)/wmax warp-wide; outputs that depend on a flagged
// step are summed sample by sample in 64 bits from NY[t] = P[t+1]-P[t] (exact, slow, never
// taken on noise-like data), all others use the 32-bit differences, which are then exact.
// RMS: the kernel also accumulates sum z^2 per (width, row, segment) -- float32 over the 8 outputs of a lane and
// step, float64 per lane along the segment, the 32 lanes added in a fixed order at the end (deterministic) --
// and, optionally, the maximum of z per (width, block of E outputs): one atomicMax per warp, width and block.
//
// Ring (per warp): slot (i mod RING) holds P[lo + i], the EXCLUSIVE prefix sum of NY (P[lo] = 0); 32-bit rings are
// stored twice (slot i and i + RING) so that reads at slot + w never wrap.  A step appends P[lo+tb .. lo+tb+WS) and
// emits the WS outputs that lag L = P.lag samples behind: o = tb - L + [0, WS).
template <class ACC, bool XF32, bool GUARD, bool RMS, bool STORE>
__global__ void __launch_bounds__(NT, MF_MINB) mf_warp_kernel(const MFParams P)
{
    static_assert(!GUARD || sizeof(ACC) == 4, "the guard belongs to the 32-bit path");
    constexpr bool MIRROR = sizeof(ACC) == 4;
    extern __shared__ __align__(16) uint8_t smem_raw[];
    const int lane = threadIdx.x & 31;
    uint8_t *wsm = smem_raw + (size_t)(threadIdx.x >> 5) * P.warp_smem;
    ACC *ring = reinterpret_cast<ACC *>(wsm);                       // [(MIRROR ? 2 : 1) * RING]
    const int RING = P.ring;
    double *dacc = reinterpret_cast<double *>(ring + (MIRROR ? 2 : 1) * RING);   // RMS: [nw][32] per-lane sums of z^2
    // RMS: [nw][32] per-lane (sum of numerator^2, maximum numerator) of the current block of E outputs
    float2 *racc = reinterpret_cast<float2 *>(dacc + (RMS ? P.nw * 32 : 0));

    const long long n = P.n;
    const int R = P.radius, L = P.lag;
    const long long N = 2ll * R + 1;
    const bool sparse = !RMS && P.sparse_list != nullptr;
    const long long item = (long long)blockIdx.x * WPB + (threadIdx.x >> 5);
    long long row, lo;
    int seg = 0, seglen, nrem, iw0 = 0, iw1 = P.nw, tb_out = 0;
    if (sparse) {
        // the block's outputs t = b*E - L + [0, E) come out of the 8 steps that start at sample b*E; the prefix sums
        // they read reach back L samples: start at the step boundary at or before b*E - L (the sums are exact
        // integers whatever the start, so z is bit-identical to the dense pass)
        if (item >= *P.sparse_count) return;
        const int2 it = P.sparse_list[item];
        iw0 = (int)(it.x / P.nrows);
        iw1 = iw0 + 1;
        row = it.x % P.nrows;
        lo = (long long)it.y * E - L;
        lo = lo < 0 ? 0 : lo / WS * WS;
        tb_out = (int)((long long)it.y * E - lo);
        nrem = (int)(n - lo);
        const long long want = (long long)tb_out - L + E;
        seglen = (int)(want < nrem ? want : nrem);
    } else {
        if (item >= P.nitems) return;
        row = P.row0 + item / P.nseg;
        seg = (int)(item % P.nseg);
        lo = (long long)seg * P.seg;
        seglen = (int)((lo + P.seg < n) ? P.seg : n - lo);
        nrem = (int)(n - lo);                  // samples from lo to the end of the row
    }
    const uint32_t *xr = reinterpret_cast<const uint32_t *>(P.x) + row * n + lo;   // sample lo of this row
    if (RMS) {
        for (int iw = 0; iw < P.nw; ++iw) {
            dacc[iw * 32 + lane] = 0.0;
            racc[iw * 32 + lane] = make_float2(0.f, -INFINITY);
        }
    }

    // ---- window sum of the sample before the segment: window start a0 = clip(lo-1-R, 0, n-N) ----
    long long a0 = lo - 1 - R;
    if (a0 < 0) a0 = 0;
    if (a0 > n - N) a0 = n - N;
    ACC carryW = 0;
    {
        const uint32_t *wb = xr + (a0 - lo);      // first sample of the window; the window is [a0, a0 + N) of the row
        ACC part = 0;
        const long long ka = (a0 + PB - 1) / PB, kb = (a0 + N) / PB;
        if (P.prefix && ka <= kb) {
            // whole blocks from the prefix sums, the two edges (< PB samples each) sample by sample
            const unsigned long long *pr = P.prefix + (size_t)row * (size_t)(P.pnb + 1);
            const int e0 = (int)(ka * PB - a0), e1 = (int)(a0 + N - kb * PB);
            for (int i = lane; i < e0; i += 32) part += (ACC)cvt_x<XF32>(__ldg(wb + i));
            const uint32_t *wt = wb + (N - e1);
            for (int i = lane; i < e1; i += 32) part += (ACC)cvt_x<XF32>(__ldg(wt + i));
            if (lane == 0) part += (ACC)(__ldg(pr + kb) - __ldg(pr + ka));
        } else {
            int head = (int)((4 - (((uintptr_t)wb >> 2) & 3)) & 3);      // scalars up to 16-byte alignment
            if (head > N) head = (int)N;
            if (lane < head) part += (ACC)cvt_x<XF32>(__ldg(wb + lane));
            const int nvec = (int)((N - head) >> 2);
            const uint4 *vb = reinterpret_cast<const uint4 *>(wb + head);
            for (int v = lane; v < nvec; v += 32) {
                const uint4 q = __ldg(vb + v);
                part += (ACC)cvt_x<XF32>(q.x) + (ACC)cvt_x<XF32>(q.y) + (ACC)cvt_x<XF32>(q.z) +
                        (ACC)cvt_x<XF32>(q.w);
            }
            const int tail = head + 4 * nvec + lane;
            if (tail < N) part += (ACC)cvt_x<XF32>(__ldg(wb + tail));
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
        carryW = part;
    }
    ACC carryP = 0;                         // P[lo] = 0: only differences are used
    // ring slots: wslot = slot of P[lo+tb] (first value written this step), rslot = slot of P[lo+tb-L] (first value
    // read this step); both stay multiples of 4 (WS, L and RING are)
    int wslot = 0;
    int rslot = (RING - L % RING) % RING;
    unsigned long long slowbits = 0;
    // d[t] = x[t+R] - x[t-R-1] while the window slides: R+1 <= t <= n-R-1, as offsets from lo
    const long long dlo_ll = (long long)R + 1 - lo;
    const int dlo = dlo_ll < -(1 << 30) ? -(1 << 30) : (int)dlo_ll;
    const int dhi = nrem - R - 1;
    // dense: z[iw][row][lo + o]; sparse: the compact block zc[item][o - (tb_out - L)]; none: RMS / maxima only
    float *const zrow = sparse ? P.zc + (size_t)item * E - (tb_out - L)
                               : (P.z ? P.z + (size_t)row * (size_t)n + (size_t)lo : nullptr);
    // register picks of the shifted streams: x[t+R] starts ra words into its first aligned vector, x[t-R-1] rb words
    const int ra = R & 3, rb = (int)((4 - ((R + 1) & 3)) & 3);
    const int last_tb = (seglen + L - 1) / WS * WS;

    for (int tb = 0; tb < seglen + L; tb += WS) {
        uint32_t dv[V], xv[V];
        // ---- this lane's 8 consecutive samples of the three streams ----
        // (steps wholly inside the clamped ends of the row -- the window does not slide there, d = 0 -- read x only;
        //  the aligned vectors of a sliding step touch up to 3 words on either side of what they need)
        const bool full = tb + WS <= nrem;        // the step lies inside the row
        const bool xin = P.vec_in && full;
        const bool slide = tb >= dlo + 3 && tb + WS - 1 + 3 <= dhi, still = tb + WS - 1 < dlo || tb > dhi;
        if (xin && (still || slide)) {
            const uint32_t *q = xr + tb + lane * V;
            const uint4 x0 = __ldg(reinterpret_cast<const uint4 *>(q)), x1 = __ldg(reinterpret_cast<const uint4 *>(q) + 1);
            const uint32_t xw[V] = {x0.x, x0.y, x0.z, x0.w, x1.x, x1.y, x1.z, x1.w};
#pragma unroll
            for (int k = 0; k < V; ++k) xv[k] = cvt_x<XF32>(xw[k]);
            if (still) {
#pragma unroll
                for (int k = 0; k < V; ++k) dv[k] = 0u;
            } else {
                const uint4 *ql = reinterpret_cast<const uint4 *>(q + (R - ra));
                const uint4 l0 = __ldg(ql), l1 = __ldg(ql + 1);
                uint4 l2 = l1;
                if (ra) l2 = __ldg(ql + 2);
                uint32_t lead[V];
                pick8(l0, l1, l2, ra, lead);
                const uint4 *qt = reinterpret_cast<const uint4 *>(q - (R + 1) - rb);
                const uint4 t0 = __ldg(qt), t1 = __ldg(qt + 1);
                uint4 t2 = t1;
                if (rb) t2 = __ldg(qt + 2);
                uint32_t trail[V];
                pick8(t0, t1, t2, rb, trail);
#pragma unroll
                for (int k = 0; k < V; ++k) dv[k] = cvt_x<XF32>(lead[k]) - cvt_x<XF32>(trail[k]);
            }
        } else {
#pragma unroll
            for (int k = 0; k < V; ++k) {
                const int o = tb + lane * V + k;
                uint32_t xt = 0, d = 0;
                if (o < nrem) {
                    xt = cvt_x<XF32>(__ldg(xr + o));
                    if (o >= dlo && o <= dhi)
                        d = cvt_x<XF32>(__ldg(xr + o + R)) - cvt_x<XF32>(__ldg(xr + o - R - 1));
                }
                xv[k] = xt;
                dv[k] = d;
            }
        }
        // ---- running window sum: scan of d ----
        ACC wv[V];
        ACC run = 0;
#pragma unroll
        for (int k = 0; k < V; ++k) {
            run += (ACC)(long long)(int)dv[k];   // d is a signed difference
            wv[k] = run;
        }
        ACC tot;
        ACC inc = warp_scan<ACC>(run, tot);
        const ACC wbase = carryW + (inc - run);
        carryW += tot;
        // ---- NY = N*x - Wsum and its exclusive prefix sum ----
        ACC pv[V];
        run = 0;
        int bad = 0;
#pragma unroll
        for (int k = 0; k < V; ++k) {
            ACC ny = (ACC)N * (ACC)xv[k] - (wbase + wv[k]);
            if (!full && tb + lane * V + k >= nrem) ny = 0;
            if (GUARD) bad |= (abs((int)ny) > P.guard_lim);
            pv[k] = run;                          // exclusive within the lane
            run += ny;
        }
        inc = warp_scan<ACC>(run, tot);
        const ACC pbase = carryP + (inc - run);
        carryP += tot;
#pragma unroll
        for (int k = 0; k < V; ++k) pv[k] += pbase;
        {
            int ws = wslot + lane * V;            // 8 consecutive slots, never across the wrap
            if (ws >= RING) ws -= RING;
            Vec8<ACC>::store(ring + ws, pv);
            if (MIRROR) Vec8<ACC>::store(ring + ws + RING, pv);
        }
        if (GUARD) slowbits = (slowbits << 1) | (__any_sync(0xffffffffu, bad) ? 1ull : 0ull);
        __syncwarp();
        // ---- outputs of the step that lags L behind (a sparse re-computation wants the block's own steps only) ----
        if (!sparse || tb >= tb_out) {
            // every boxcar of this step's outputs is complete (only steps at the end of a ROW are not); outputs before
            // the segment (first step: the lag) or past it (last step) are masked per group of four
            const bool complete = tb + WS - 1 <= nrem;
            constexpr bool store = STORE;
            const bool slow = GUARD && (slowbits & P.guard_hist);
            if (MIRROR && complete && !slow && P.vec_out) {
                const int oa = tb - L + 4 * lane, ob4 = oa + 4 * 32;
                const bool va = oa >= 0 && oa + 4 <= seglen, vb = ob4 >= 0 && ob4 + 4 <= seglen;
                // ---- vector path: lane = 2 x 4 consecutive outputs; ring read and z written 128 bits at a time ----
                int s0 = rslot + 4 * lane, s1 = s0 + 4 * 32;
                if (s0 >= RING) s0 -= RING;
                if (s1 >= RING) s1 -= RING;
                const uint4 pa = *reinterpret_cast<const uint4 *>(ring + s0), pb = *reinterpret_cast<const uint4 *>(ring + s1);
                float *const zp0 = zrow + (tb - L) + 4 * lane;
                // two passes over the widths: multiples of 4 first (the ring vectors are the operands), then the
                // others (two vectors + a register pick) -- one loop would make the compiler funnel both through
                // the same registers with eight moves per width
#pragma unroll 1
                for (int pass = 0; pass < 2; ++pass) {
#pragma unroll 1
                    // (the host lists the widths that are multiples of 4 first: wl[0 .. n4), then the others)
                    for (int q = pass ? P.n4 : 0; q < (pass ? P.nw : P.n4); ++q) {
                        const int iw = P.wl[q];
                        if (sparse && iw != iw0) continue;
                        const int w = P.w[iw], wa = w & 3, wo = w - wa;
                        float fa[4], fb[4];     // float32 of the exact integer numerators
                        const uint4 a0v = *reinterpret_cast<const uint4 *>(ring + s0 + wo);
                        const uint4 b0v = *reinterpret_cast<const uint4 *>(ring + s1 + wo);
                        if (pass == 0) {
                            fa[0] = acc_to_float((uint32_t)(a0v.x - pa.x)); fa[1] = acc_to_float((uint32_t)(a0v.y - pa.y));
                            fa[2] = acc_to_float((uint32_t)(a0v.z - pa.z)); fa[3] = acc_to_float((uint32_t)(a0v.w - pa.w));
                            fb[0] = acc_to_float((uint32_t)(b0v.x - pb.x)); fb[1] = acc_to_float((uint32_t)(b0v.y - pb.y));
                            fb[2] = acc_to_float((uint32_t)(b0v.z - pb.z)); fb[3] = acc_to_float((uint32_t)(b0v.w - pb.w));
                        } else {
                            const uint4 a1v = *reinterpret_cast<const uint4 *>(ring + s0 + wo + 4);
                            const uint4 b1v = *reinterpret_cast<const uint4 *>(ring + s1 + wo + 4);
                            uint32_t qa[4], qb[4];
                            pick4(a0v, a1v, wa, qa);
                            pick4(b0v, b1v, wa, qb);
                            fa[0] = acc_to_float((uint32_t)(qa[0] - pa.x)); fa[1] = acc_to_float((uint32_t)(qa[1] - pa.y));
                            fa[2] = acc_to_float((uint32_t)(qa[2] - pa.z)); fa[3] = acc_to_float((uint32_t)(qa[3] - pa.w));
                            fb[0] = acc_to_float((uint32_t)(qb[0] - pb.x)); fb[1] = acc_to_float((uint32_t)(qb[1] - pb.y));
                            fb[2] = acc_to_float((uint32_t)(qb[2] - pb.z)); fb[3] = acc_to_float((uint32_t)(qb[3] - pb.w));
                        }
                        if (RMS) {
                            float2 st = racc[iw * 32 + lane];
                            if (va) {
#pragma unroll
                                for (int i = 0; i < 4; ++i) { st.x = __fmaf_rn(fa[i], fa[i], st.x); st.y = fmaxf(st.y, fa[i]); }
                            }
                            if (vb) {
#pragma unroll
                                for (int i = 0; i < 4; ++i) { st.x = __fmaf_rn(fb[i], fb[i], st.x); st.y = fmaxf(st.y, fb[i]); }
                            }
                            racc[iw * 32 + lane] = st;
                        }
                        if (store) {
                            const float scl = P.scale[iw];
                            float *zp = zp0 + (long long)iw * P.plane;
                            if (va)
                                __stcs(reinterpret_cast<float4 *>(zp), make_float4(fa[0] * scl, fa[1] * scl, fa[2] * scl, fa[3] * scl));
                            if (vb)
                                __stcs(reinterpret_cast<float4 *>(zp + 4 * 32),
                                       make_float4(fb[0] * scl, fb[1] * scl, fb[2] * scl, fb[3] * scl));
                        }
                    }
                }
            } else {
                // ---- scalar path: lane = outputs o = tb - L + lane + 32 k ----
                const int ob = tb - L + lane;
                for (int iw = iw0; iw < iw1; ++iw) {
                    float *zp = zrow + ob + (long long)iw * P.plane;
                    const int w = P.w[iw];
                    const float scl = P.scale[iw];
                    const int lim = nrem - w;                 // t + w <= n  <=>  o <= lim
                    float ss = 0.f, mx = -INFINITY;
#pragma unroll 1
                    for (int k = 0; k < V; ++k) {
                        const int o = ob + k * 32;
                        if (o < 0 || o >= seglen) continue;
                        int sl = rslot + lane + k * 32;
                        if (sl >= RING) sl -= RING;
                        float f = 0.f;                        // float32 of the exact integer numerator
                        if (o <= lim) {
                            if (slow) {
                                long long zz = 0;
                                uint32_t prev = (uint32_t)ring[sl];
                                for (int q = 0; q < w; ++q) {
                                    if (++sl >= RING) sl = 0;
                                    const uint32_t cur = (uint32_t)ring[sl];
                                    zz += (long long)(int)(cur - prev);
                                    prev = cur;
                                }
                                f = (float)zz;
                            } else {
                                int s2 = sl + w;
                                if (!MIRROR && s2 >= RING) s2 -= RING;
                                f = acc_to_float((ACC)(ring[s2] - ring[sl]));
                            }
                        }
                        if (RMS) { ss = __fmaf_rn(f, f, ss); mx = fmaxf(mx, f); }
                        if (store) __stcs(zp + k * 32, f * scl);   // streaming store: keep x, not z, in L2
                    }
                    if (RMS) {
                        float2 st = racc[iw * 32 + lane];
                        st.x += ss;
                        st.y = fmaxf(st.y, mx);
                        racc[iw * 32 + lane] = st;
                    }
                }
            }
            // the outputs of this step are t = lo + tb - L + [0, WS): block (lo + tb) / E of the hint.  When the block
            // (or the segment) ends: the lane sums of numerator^2 (float32 over <= 64 outputs) go into the float64 sums
            // scaled to z^2, the lane maxima into the block maximum -- neighbouring segments share a block: atomicMax
            if (RMS && ((tb + WS) % E == 0 || tb == last_tb)) {
                __syncwarp();
                for (int iw = 0; iw < P.nw; ++iw) {
                    const float2 st = racc[iw * 32 + lane];
                    const double scl = (double)P.scale[iw];
                    dacc[iw * 32 + lane] += (double)st.x * (scl * scl);
                    racc[iw * 32 + lane] = make_float2(0.f, -INFINITY);
                    if (P.blockmax) {
                        // max z = fl(max numerator * scale): both roundings are monotone
                        const int m = __reduce_max_sync(0xffffffffu, ordered_int(st.y * P.scale[iw]));
                        if (lane == 0)
                            atomicMax(P.blockmax + ((size_t)iw * P.nrows + (size_t)row) * P.nblk + (lo + tb) / E, m);
                    }
                }
            }
        }
        wslot += WS;
        if (wslot >= RING) wslot -= RING;
        rslot += WS;
        if (rslot >= RING) rslot -= RING;
        __syncwarp();
    }
    if (RMS) {
        // the 32 lane sums of each width, added in a fixed order (shuffle tree): deterministic
        for (int iw = 0; iw < P.nw; ++iw) {
            double v = dacc[iw * 32 + lane];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
            if (lane == 0) P.partial[((size_t)iw * (size_t)P.nrows + (size_t)row) * P.nseg + seg] = v;
        }
    }
}

// prefix[row][k] = sum of x[row][0 .. min(k * PB, n)), k = 0 .. pnb (64-bit: exact; 32-bit users take it mod 2^32).
// One CTA of 8 warps per row; a warp sums one block of PB = 256 samples at a time (8 consecutive samples per lane,
// 128-bit loads where the row allows), the block sums of up to 2048 blocks are gathered in shared memory and
// scanned by the CTA, with a carry across such chunks for very long rows.  Reads x once: HBM-bound.
template <bool XF32>
__global__ void __launch_bounds__(256) mf_prefix_kernel(const uint32_t *__restrict__ x, long long n, int pnb,
                                                        unsigned long long *__restrict__ prefix, int vec, long long row0)
{
    constexpr int CHUNK = 2048;
    __shared__ unsigned long long sb[CHUNK];
    __shared__ unsigned long long swarp[8];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t *xr = x + (size_t)(row0 + blockIdx.x) * (size_t)n;
    unsigned long long *pr = prefix + (size_t)(row0 + blockIdx.x) * (size_t)(pnb + 1);
    unsigned long long carry = 0;
    for (int k0 = 0; k0 < pnb; k0 += CHUNK) {
        const int nk = pnb - k0 < CHUNK ? pnb - k0 : CHUNK;
        for (int k = warp; k < nk; k += 8) {
            const long long t = (long long)(k0 + k) * PB + lane * 8;
            unsigned long long v = 0;
            if (vec && t + 8 <= n) {
                const uint4 a = __ldg(reinterpret_cast<const uint4 *>(xr + t)), b = __ldg(reinterpret_cast<const uint4 *>(xr + t) + 1);
                v = (unsigned long long)cvt_x<XF32>(a.x) + cvt_x<XF32>(a.y) + cvt_x<XF32>(a.z) + cvt_x<XF32>(a.w) +
                    cvt_x<XF32>(b.x) + cvt_x<XF32>(b.y) + cvt_x<XF32>(b.z) + cvt_x<XF32>(b.w);
            } else {
                for (int i = 0; i < 8; ++i)
                    if (t + i < n) v += cvt_x<XF32>(__ldg(xr + t + i));
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            if (lane == 0) sb[k] = v;
        }
        __syncthreads();
        // exclusive scan of sb[0 .. nk): 8 consecutive entries per thread
        unsigned long long loc[8], run = 0;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const int k = threadIdx.x * 8 + i;
            loc[i] = run;
            run += k < nk ? sb[k] : 0ull;
        }
        unsigned long long inc = run;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const unsigned long long u = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += u;
        }
        if (lane == 31) swarp[warp] = inc;
        __syncthreads();
        unsigned long long base = carry, tot = 0;
        for (int q = 0; q < 8; ++q) {
            if (q < warp) base += swarp[q];
            tot += swarp[q];
        }
        base += inc - run;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const int k = threadIdx.x * 8 + i;
            if (k < nk) pr[k0 + k] = base + loc[i];
        }
        carry += tot;
        __syncthreads();
    }
    if (threadIdx.x == 0) pr[pnb] = carry;
}

// rms[s] = fl32( sqrt( (sum of the nseg partials of series s, in order) / n ) )
__global__ void mf_rms_finish_kernel(const double *__restrict__ partial, long long nseries, int nseg, long long n,
                                     float *__restrict__ rms)
{
    const long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= nseries) return;
    double t = 0.0;
    for (int q = 0; q < nseg; ++q) t += partial[s * nseg + q];
    rms[s] = (float)sqrt(t / (double)n);
}

}  // namespace

// Samples per work item (one warp): a multiple of E.  With the per-row prefix sums the start of an item is cheap, so
// segments are short: the items of a row then run at the same time (consecutive items = consecutive segments of a
// row), the rows in flight -- resident warps / segments per row -- fit L2, and the x[t - R - 1] and x[t] streams are
// served from the lines the x[t + R] stream brought in (profiles/r2_matched_filter.md).  Depends only on nsamps, so
// that the workspace size can be computed ahead of the call.
#ifndef MF_WSEG
#define MF_WSEG (2 * E)
#endif
long long mf_warp_segment(long long nrows, long long nsamps)
{
    (void)nrows;
    long long seg = MF_WSEG;
    if (seg > nsamps) seg = (nsamps + E - 1) / E * E;
    return seg;
}

size_t mf_warp_workspace_bytes(long long nrows, long long nsamps, int nwidths)
{
    const long long seg = mf_warp_segment(nrows, nsamps), nseg = (nsamps + seg - 1) / seg;
    const long long pnb = (nsamps + PB - 1) / PB;
    return (size_t)nwidths * (size_t)nrows * (size_t)nseg * sizeof(double) + (size_t)nrows * (size_t)(pnb + 1) * 8;
}

// sparse_list / sparse_count / zc / max_blocks: the sparse re-computation of dedisp_search_events (one CTA per listed
// block, z_dev and rms_dev null); otherwise the dense pass (z_dev may be null when rms_dev is given: RMS and block
// maxima only).
dedisp_status mf_warp_run(const void *x_dev, dedisp_out_dtype x_dtype, long long nrows, long long nsamps, int radius,
                     const int *widths_host, int nwidths, unsigned int x_max, float *z_dev, float *rms_dev,
                     int *blockmax_dev, void *workspace_dev, size_t workspace_bytes, void *cuda_stream,
                     const int2 *sparse_list, const int *sparse_count, float *zc, long long max_blocks)
{
    // workspace (dense with rms_dev, and sparse): [nwidths * nrows * nseg doubles: partial sums of z^2][nrows * (pnb + 1)
    // uint64: per-row prefix sums of x]; mf_warp_workspace_bytes().  The sparse pass re-uses the prefix sums the RMS
    // pass of the same dedisp_search_events call left there.  Without a workspace (workspace_dev null) every work item
    // sums its first window sample by sample.
    const bool sparse = sparse_list != nullptr;
    if (!x_dev || !widths_host || nrows < 1 || nsamps < 1 || radius < 0) return DEDISP_ERR_INVALID_ARG;
    if (sparse ? (!sparse_count || !zc || max_blocks < 1 || max_blocks > 0x7fffffffll || z_dev || rms_dev)
               : (!z_dev && !rms_dev))
        return DEDISP_ERR_INVALID_ARG;
    if (x_dtype != DEDISP_OUT_U32 && x_dtype != DEDISP_OUT_F32) return DEDISP_ERR_UNSUPPORTED_DTYPE;
    if (nwidths < 1 || nwidths > MAXW || nsamps > (1ll << 30)) return DEDISP_ERR_INVALID_ARG;
    if (((uintptr_t)x_dev & 3u) || ((uintptr_t)z_dev & 3u) || ((uintptr_t)zc & 3u)) return DEDISP_ERR_INVALID_ARG;
    const long long N = 2ll * radius + 1;
    if (N > nsamps) return DEDISP_ERR_INVALID_ARG;
    if (x_max == 0) x_max = (1u << 24) - 1;
    if (x_max >= (1u << 24)) return DEDISP_ERR_OVERFLOW;
    MFParams P;
    P.x = x_dev;
    P.z = z_dev;
    P.nrows = nrows;
    P.n = nsamps;
    P.radius = radius;
    P.nw = nwidths;
    P.wmax = 0;
    for (int i = 0; i < nwidths; ++i) {
        const int w = widths_host[i];
        if (w < 1 || w > nsamps || w > DEDISP_MF_MAX_WIDTH) return DEDISP_ERR_INVALID_ARG;
        P.w[i] = w;
        P.scale[i] = (float)(1.0 / ((double)N * std::sqrt((double)w)));
        if (w > P.wmax) P.wmax = w;
    }
    for (int i = nwidths; i < MAXW; ++i) { P.w[i] = 1; P.scale[i] = 0.f; }
    P.n4 = 0;
    for (int i = 0; i < nwidths; ++i)
        if (P.w[i] % 4 == 0) P.wl[P.n4++] = i;
    for (int i = 0, q = P.n4; i < nwidths; ++i)
        if (P.w[i] % 4 != 0) P.wl[q++] = i;
    for (int i = nwidths; i < MAXW; ++i) P.wl[i] = 0;
    P.lag = P.wmax;       // (the hint geometry of dedisp_matched_filter_hint_blocks: outputs trail by the largest width)
    const int ring = (WS + P.lag + 8 + 7) & ~7;
    P.ring = ring;
    const bool rows16 = nsamps % 4 == 0;
    P.vec_in = rows16 && ((uintptr_t)x_dev & 15u) == 0;
    // 128-bit ring reads / stores need the lag to be a multiple of 4 (else the scalar path serves every step)
    P.vec_out = (P.lag % 4 == 0) && (sparse ? 1 : (z_dev ? (rows16 && ((uintptr_t)z_dev & 15u) == 0) : 1));
    const long long seg = mf_warp_segment(nrows, nsamps);
    P.seg = (int)seg;
    const long long nseg = (nsamps + seg - 1) / seg;
    P.nseg = (int)nseg;
    P.nitems = nrows * nseg;
    P.row0 = 0;
    P.plane = sparse ? 0 : nrows * nsamps;
    if (nrows * nseg > 0x7fffffffll) return DEDISP_ERR_INVALID_ARG;
    // |boxcar numerator| <= wmax * N * x_max must fit the signed accumulator
    const long double bound = (long double)P.wmax * (long double)N * (long double)x_max;
    if (bound >= 9.0e18L) return DEDISP_ERR_OVERFLOW;
    // 32-bit words when every boxcar provably fits; guarded 32-bit words when at least NY does
    // (N*x_max < 2^31); 64-bit words otherwise
    const bool fits32 = bound < 2147483648.0L;
    const bool guard = !fits32 && (long double)N * (long double)x_max < 2147483648.0L;
    const bool wide = !fits32 && !guard;
    P.guard_lim = (int)(2147483647ll / P.wmax);
    {   // outputs of a step read prefix sums of this step and of the ceil(L / WS) steps before it (<= 33 + 1 flags)
        const int nflags = (P.lag + WS - 1) / WS + 1;
        P.guard_hist = nflags >= 64 ? ~0ull : ((1ull << nflags) - 1ull);
    }
    const size_t accb = wide ? 8 : 4;
    const bool rms = rms_dev != nullptr;
    P.partial = (double *)workspace_dev;
    const long long pnb = (nsamps + PB - 1) / PB;
    const size_t partial_bytes = (size_t)nwidths * (size_t)nrows * (size_t)nseg * sizeof(double);
    const bool have_ws = workspace_dev && ((uintptr_t)workspace_dev & 7u) == 0 &&
                         workspace_bytes >= partial_bytes + (size_t)nrows * (size_t)(pnb + 1) * 8;
    P.prefix = have_ws ? (const unsigned long long *)((const uint8_t *)workspace_dev + partial_bytes) : nullptr;
    P.pnb = (int)pnb;
    P.blockmax = blockmax_dev;
    P.nblk = (int)((nsamps + P.lag + E - 1) / E);
    P.sparse_list = sparse_list;
    P.sparse_count = sparse_count;
    P.zc = zc;
    if (blockmax_dev && (!rms || ((uintptr_t)blockmax_dev & 3u))) return DEDISP_ERR_INVALID_ARG;
    if (rms) {
        if (!workspace_dev || ((uintptr_t)workspace_dev & 7u) || ((uintptr_t)rms_dev & 3u) ||
            workspace_bytes < partial_bytes)
            return DEDISP_ERR_INVALID_ARG;
    }
    const size_t warp_smem = ((wide ? 1 : 2) * (size_t)ring * accb + (rms ? (size_t)nwidths * 32 * 16 : 0) + 15) &
                             ~(size_t)15;
    P.warp_smem = (int)warp_smem;
    const size_t smem = WPB * warp_smem;
    if (smem > 227 * 1024) return DEDISP_ERR_INVALID_ARG;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    if (nrows > 0x7fffffffll) return DEDISP_ERR_INVALID_ARG;
    cudaError_t e = cudaSuccess;
    if (blockmax_dev &&   // every byte 0x80: below the image of any finite float
        cudaMemsetAsync(blockmax_dev, 0x80, (size_t)nwidths * (size_t)nrows * (size_t)P.nblk * 4, s) != cudaSuccess)
        return DEDISP_ERR_CUDA;
    // Dense passes with prefix sums can run in blocks of rows whose x fits L2 (MF_L2_ROW_BYTES: the prefix kernel of a
    // block brings its rows in, the filter kernel of the block then reads them from L2).  Measured on the gulp it
    // LOSES (search step 0.495 ms in one launch, 0.616 / 0.666 / 0.838 ms with 110 / 80 / 40 MB blocks): the filter
    // kernel is bound by instruction issue and latency per work item, not by DRAM, and every launch pays its own
    // ramp and tail.  The default is therefore one launch; the knob stays for other shapes.
#ifndef MF_L2_ROW_BYTES
#define MF_L2_ROW_BYTES (1ll << 50)
#endif
    long long rows_per_launch = nrows;
    if (P.prefix && !sparse) {
        rows_per_launch = MF_L2_ROW_BYTES / (nsamps * 4);
        if (rows_per_launch < 64) rows_per_launch = 64;
        if (rows_per_launch > nrows) rows_per_launch = nrows;
    }
    const bool f32 = (x_dtype == DEDISP_OUT_F32);
#define MF_LAUNCH1(ACC, F, G, R, ST)                                                                  \
    do {                                                                                             \
        e = cudaFuncSetAttribute(mf_warp_kernel<ACC, F, G, R, ST>,                            \
                                 cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);            \
        if (e == cudaSuccess) mf_warp_kernel<ACC, F, G, R, ST><<<grid, block, smem, s>>>(P);  \
    } while (0)
#define MF_LAUNCH(ACC, F, G)                               \
    do {                                                   \
        if (rms && z_dev) MF_LAUNCH1(ACC, F, G, true, true);   \
        else if (rms) MF_LAUNCH1(ACC, F, G, true, false);  \
        else MF_LAUNCH1(ACC, F, G, false, true);           \
    } while (0)
    for (long long r0 = 0; r0 < nrows && e == cudaSuccess; r0 += rows_per_launch) {
        const long long nr = nrows - r0 < rows_per_launch ? nrows - r0 : rows_per_launch;
        if (P.prefix && !sparse) {
            // per-row prefix sums of x for the cheap start of every work item (the sparse pass re-uses them)
            unsigned long long *pw = const_cast<unsigned long long *>(P.prefix);
            const int pvec = rows16 && ((uintptr_t)x_dev & 15u) == 0;
            if (f32)
                mf_prefix_kernel<true><<<(unsigned)nr, 256, 0, s>>>((const uint32_t *)x_dev, nsamps, P.pnb, pw, pvec, r0);
            else
                mf_prefix_kernel<false><<<(unsigned)nr, 256, 0, s>>>((const uint32_t *)x_dev, nsamps, P.pnb, pw, pvec, r0);
            if (cudaGetLastError() != cudaSuccess) return DEDISP_ERR_CUDA;
            ++g_launch_count;
        }
        P.row0 = r0;
        P.nitems = nr * nseg;
        const dim3 grid((unsigned)(((sparse ? max_blocks : nr * nseg) + WPB - 1) / WPB)), block(NT);
        if (wide) {
            if (f32) MF_LAUNCH(unsigned long long, true, false);
            else MF_LAUNCH(unsigned long long, false, false);
        } else if (guard) {
            if (f32) MF_LAUNCH(uint32_t, true, true);
            else MF_LAUNCH(uint32_t, false, true);
        } else {
            if (f32) MF_LAUNCH(uint32_t, true, false);
            else MF_LAUNCH(uint32_t, false, false);
        }
        if (e == cudaSuccess) e = cudaGetLastError();
        if (e == cudaSuccess) ++g_launch_count;
    }
#undef MF_LAUNCH
#undef MF_LAUNCH1
    if (e != cudaSuccess) return DEDISP_ERR_CUDA;
    if (rms) {
        const long long nseries = (long long)nwidths * nrows;
        mf_rms_finish_kernel<<<(unsigned)((nseries + 255) / 256), 256, 0, s>>>(P.partial, nseries, P.nseg, nsamps, rms_dev);
        if (cudaGetLastError() != cudaSuccess) return DEDISP_ERR_CUDA;
        ++g_launch_count;
    }
    return DEDISP_OK;
}
