// matched_filter.cu -- baseline removal by running mean + boxcar matched filters
// (Sec. 2.3), one streaming pass over
// the dedispersed time series, HBM-bound.
//
//   y[t]   = x[t] - (1/N) sum_{k=a(t)}^{a(t)+N-1} x[k],  N = 2R+1, a(t) = clip(t-R, 0, n-N)
//   z_w[t] = (1/sqrt(w)) sum_{k<w} y[t+k]   for t <= n-w,   0 beyond
//
// The paper's algorithm is "prefix sum, then subtract the points at plus and minus
// the window radius", and the same again for the boxcars.  Here both prefix sums are
// block-local scans carried along a row segment, in exact modular integers:
//   Wsum[t] = Wsum[t-1] + (x[t+R] - x[t-R-1])           (running window sum, scan of d)
//   NY[t]   = N*x[t] - Wsum[t]                           (N * baseline-removed sample)
//   P[t+1]  = P[t] + NY[t]                               (prefix sum of NY, kept in a ring)
//   z_w[t]  = float(P[t+w] - P[t]) * fl32(1 / (N sqrt(w)))
// Differences of modular prefix sums are exact as long as the true value fits the
// word, so 32-bit words serve whenever wmax*N*x_max < 2^31 (or, guarded by a per-step
// check of the data, whenever N*x_max < 2^31) and 64-bit words otherwise.
// A work item is (row, segment of SEG samples); a CTA walks its segment in steps of
// E = NT*V samples: coalesced loads of the three input streams (x[t], x[t+R],
// x[t-R-1]; the two trailing streams hit L2), two block scans, then the outputs of
// the step that lags wmax samples behind, written with coalesced 4-byte stores.
#include <cmath>
#include <cstdlib>
#include <type_traits>

#include "dedisp_internal.h"

// resident CTAs per SM the register budget is set for (measured on the gulp, 7 widths: plain kernel
// 4 / 5 / 6 CTAs = 0.534 / 0.526 / 0.626 ms; with the fused sum of squares 0.925 / 1.000 / 1.010 ms per
// matched_filter_rms + find_events step)
#ifndef MF_MINB
#define MF_MINB 5
#endif
#ifndef MF_MINB_RMS
#define MF_MINB_RMS 4
#endif

namespace {

constexpr int NT = 256;          // threads per CTA
constexpr int V = 8;             // samples per thread per step
constexpr int E = NT * V;        // samples per step
constexpr int MAXW = 16;         // boxcar widths per call

struct MFParams {
    const void *x;               // [nrows][n] uint32 or float32 (exact integers)
    float *z;                    // [nw][nrows][n]
    long long nrows, n;
    int radius;
    int nw;
    int wmax;
    int ring;                    // ring entries, multiple of 8, >= E + wmax + 1
    int seg;                     // samples per segment (multiple of E)
    int nseg;
    int guard_lim;               // guarded 32-bit mode: |NY| <= guard_lim => every boxcar fits int32
    int guard_hist;              // mask of the step flags the outputs of one step depend on
    int w[MAXW];
    float scale[MAXW];           // fl32(1 / (N sqrt(w)))
    double *partial;             // RMS variant: [nw][nrows][nseg] sums of z^2 over a segment
    int *blockmax;               // RMS variant, optional: [nw][nrows][nblk] upper bounds of z per block of E outputs
    int nblk;
};

// inclusive block scan of one value per thread; returns the thread's inclusive prefix and
// the block total.  sc: NT/32 words of shared scratch.
template <class ACC>
__device__ __forceinline__ ACC block_scan(ACC v, ACC *sc, ACC &total)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        ACC u = __shfl_up_sync(0xffffffffu, v, o);
        if (lane >= o) v += u;
    }
    if (lane == 31) sc[warp] = v;
    __syncthreads();
    // the NT/32 = 8 warp totals: every lane takes one (lane & 7), an 8-wide shuffle scan gives the
    // exclusive prefix of this thread's warp and the block total
    const ACC mine = sc[lane & (NT / 32 - 1)];
    ACC inc = mine;
#pragma unroll
    for (int o = 1; o < NT / 32; o <<= 1) {
        const ACC u = __shfl_up_sync(0xffffffffu, inc, o, NT / 32);
        if ((lane & (NT / 32 - 1)) >= o) inc += u;
    }
    const ACC base = __shfl_sync(0xffffffffu, inc - mine, warp, NT / 32);
    const ACC tot = __shfl_sync(0xffffffffu, inc, NT / 32 - 1, NT / 32);
    total = tot;
    __syncthreads();
    return v + base;
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

// Push a thread's maximum of z over the outputs of one step into blockmax (see dedisp.h: hint of
// dedisp_find_events_hinted): order-preserving int image of the float, warp maximum, one atomicMax.
__device__ __forceinline__ void push_block_max(int *dst, float mx)
{
    int o = __float_as_int(mx);
    o = o >= 0 ? o : o ^ 0x7fffffff;
    o = __reduce_max_sync(0xffffffffu, o);
    if ((threadIdx.x & 31) == 0) atomicMax(dst, o);
}

// GUARD (32-bit words only, host has checked N*x_max < 2^31 so that NY is exact in int32):
// the worst-case boxcar wmax*N*x_max does not fit 32 bits, but real series stay far below
// it.  Every step flags |NY| > (2^31-1)/wmax block-wide; outputs that depend on a flagged
// step are summed sample by sample in 64 bits from NY[t] = P[t+1]-P[t] (exact, slow, never
// taken on noise-like data), all others use the 32-bit differences, which are then exact.
// RMS: the kernel also accumulates sum z^2 per (width, row, segment) -- float32 per thread over the
// <= 64 outputs it writes per width and segment, then float64 across the block in a fixed order --
// so that the noise level of every filtered series is known without reading z back.
template <class ACC, bool XF32, bool GUARD, bool RMS>
__global__ void __launch_bounds__(NT, RMS ? MF_MINB_RMS : MF_MINB) matched_filter_kernel(const MFParams P)
{
    static_assert(!GUARD || sizeof(ACC) == 4, "the guard belongs to the 32-bit path");
    // 32-bit rings are stored twice (slot i and i+RING) so that reads at slot+w never wrap;
    // 64-bit rings are not (the doubled footprint costs more occupancy than the wrap test)
    constexpr bool MIRROR = sizeof(ACC) == 4;
    int slowbits = 0;
    extern __shared__ __align__(16) uint8_t smem_raw[];
    uint32_t *sX = reinterpret_cast<uint32_t *>(smem_raw);          // [E]  x[t]
    uint32_t *sD = sX + E;                                          // [E]  x[t+R] - x[t-R-1]
    ACC *sc = reinterpret_cast<ACC *>(sD + E);                      // [NT/32]
    ACC *ring = sc + NT / 32;                                       // [2*ring] slot i (and i+ring) holds P[i+1]
    const int RING = P.ring;                                        // multiple of 8, >= E + wmax + 1
    float *sAcc = reinterpret_cast<float *>(ring + (MIRROR ? 2 : 1) * RING);   // RMS: [nw][NT]
    if (RMS)
        for (int iw = 0; iw < P.nw; ++iw) sAcc[iw * NT + threadIdx.x] = 0.f;

    const long long row = blockIdx.x / P.nseg;
    const int seg = (int)(blockIdx.x % P.nseg);
    const long long n = P.n;
    const int R = P.radius;
    const long long N = 2ll * R + 1;
    const long long lo = (long long)seg * P.seg;
    const int seglen = (int)((lo + P.seg < n) ? P.seg : n - lo);
    const int nrem = (int)(n - lo);                  // samples from lo to the end of the row
    const uint32_t *xr = reinterpret_cast<const uint32_t *>(P.x) + row * n + lo;   // sample lo of this row
    const int j = threadIdx.x;

    // ---- window sum of the sample before the segment: window start a0 = clip(lo-1-R, 0, n-N) ----
    long long a0 = lo - 1 - R;
    if (a0 < 0) a0 = 0;
    if (a0 > n - N) a0 = n - N;
    ACC part = 0;
    {
        const uint32_t *wb = xr + (a0 - lo);
        int head = (int)((4 - (((uintptr_t)wb >> 2) & 3)) & 3);      // scalars up to 16-byte alignment
        if (head > N) head = (int)N;
        if (j < head) part += (ACC)cvt_x<XF32>(__ldg(wb + j));
        const int nvec = (int)((N - head) >> 2);
        const uint4 *vb = reinterpret_cast<const uint4 *>(wb + head);
        for (int v = j; v < nvec; v += NT) {
            const uint4 q = __ldg(vb + v);
            part += (ACC)cvt_x<XF32>(q.x) + (ACC)cvt_x<XF32>(q.y) + (ACC)cvt_x<XF32>(q.z) +
                    (ACC)cvt_x<XF32>(q.w);
        }
        const int tail = head + 4 * nvec + j;
        if (tail < N) part += (ACC)cvt_x<XF32>(__ldg(wb + tail));
    }
    ACC carryW;
    block_scan<ACC>(part, sc, carryW);
    ACC carryP = 0;                         // P[lo] = 0: only differences are used
    // ring slots: wslot = slot of P[lo+tb+1] (first value written this step),
    //             rslot = slot of P[lo+tb-wmax] (first value read this step)
    int wslot = (int)(lo % RING);
    int rslot = wslot - 1 - P.wmax;
    if (rslot < 0) rslot += RING;
    if (j == 0) {
        const int s0 = wslot == 0 ? RING - 1 : wslot - 1;
        ring[s0] = 0;
        if (MIRROR) ring[s0 + RING] = 0;
    }
    // d[t] = x[t+R] - x[t-R-1] while the window slides: R+1 <= t <= n-R-1, as offsets from lo
    const long long dlo_ll = (long long)R + 1 - lo;
    const int dlo = dlo_ll < -(1 << 30) ? -(1 << 30) : (int)dlo_ll;
    const int dhi = nrem - R - 1;
    const size_t plane = (size_t)P.nrows * (size_t)n;
    float *const zrow = P.z + (size_t)row * (size_t)n + (size_t)lo;

    for (int tb = 0; tb < seglen + P.wmax; tb += E) {
        // ---- the three input streams, coalesced (the two trailing ones hit L2) ----
        if (tb + E <= nrem && tb >= dlo && tb + E - 1 <= dhi) {
#pragma unroll
            for (int k = 0; k < V; ++k) {
                const int i = j + k * NT;
                const uint32_t *q = xr + tb + i;
                sX[i] = cvt_x<XF32>(__ldg(q));
                sD[i] = cvt_x<XF32>(__ldg(q + R)) - cvt_x<XF32>(__ldg(q - R - 1));
            }
        } else {
#pragma unroll
            for (int k = 0; k < V; ++k) {
                const int i = j + k * NT;
                const int o = tb + i;
                uint32_t xt = 0, d = 0;
                if (o < nrem) {
                    xt = cvt_x<XF32>(__ldg(xr + o));
                    if (o >= dlo && o <= dhi)
                        d = cvt_x<XF32>(__ldg(xr + o + R)) - cvt_x<XF32>(__ldg(xr + o - R - 1));
                }
                sX[i] = xt;
                sD[i] = d;
            }
        }
        __syncthreads();
        // ---- running window sum: scan of d (8 consecutive samples per thread) ----
        uint32_t dv[V], xv[V];
        *reinterpret_cast<uint4 *>(&dv[0]) = reinterpret_cast<const uint4 *>(sD + j * V)[0];
        *reinterpret_cast<uint4 *>(&dv[4]) = reinterpret_cast<const uint4 *>(sD + j * V)[1];
        *reinterpret_cast<uint4 *>(&xv[0]) = reinterpret_cast<const uint4 *>(sX + j * V)[0];
        *reinterpret_cast<uint4 *>(&xv[4]) = reinterpret_cast<const uint4 *>(sX + j * V)[1];
        ACC wv[V];
        ACC run = 0;
#pragma unroll
        for (int k = 0; k < V; ++k) {
            run += (ACC)(long long)(int)dv[k];   // d is a signed difference
            wv[k] = run;
        }
        ACC tot;
        ACC inc = block_scan<ACC>(run, sc, tot);
        const ACC wbase = carryW + (inc - run);
        carryW += tot;
        // ---- NY = N*x - Wsum and its prefix sum ----
        ACC pv[V];
        run = 0;
        int bad = 0;
#pragma unroll
        for (int k = 0; k < V; ++k) {
            ACC ny = (ACC)N * (ACC)xv[k] - (wbase + wv[k]);
            if (tb + j * V + k >= nrem) ny = 0;
            if (GUARD) bad |= (abs((int)ny) > P.guard_lim);
            run += ny;
            pv[k] = run;
        }
        inc = block_scan<ACC>(run, sc, tot);
        const ACC pbase = carryP + (inc - run);
        carryP += tot;
#pragma unroll
        for (int k = 0; k < V; ++k) pv[k] += pbase;
        {
            int ws = wslot + j * V;               // 8 consecutive slots, never across the wrap
            if (ws >= RING) ws -= RING;
            Vec8<ACC>::store(ring + ws, pv);
            if (MIRROR) Vec8<ACC>::store(ring + ws + RING, pv);
        }
        if (GUARD) slowbits = (slowbits << 1) | (__syncthreads_or(bad) ? 1 : 0);
        else __syncthreads();
        // ---- outputs of the step that lags wmax behind: o = tb - wmax + j + k*NT ----
        const int ob = tb - P.wmax + j;
        int rs[V];
        ACC p0[V];
#pragma unroll
        for (int k = 0; k < V; ++k) {
            int sl = rslot + j + k * NT;
            if (sl >= RING) sl -= RING;
            rs[k] = sl;
            p0[k] = ring[sl];
        }
        const bool interior = (tb - P.wmax >= 0) && (tb - P.wmax + E <= seglen) &&
                              (tb + E - 1 <= nrem);      // every output valid, every boxcar complete
        float *zp = zrow + ob;
        // outputs of this step are t = lo + tb - wmax + [0, E): block (lo + tb) / E of the hint
        int *const bmax = (RMS && P.blockmax) ? P.blockmax + (size_t)row * P.nblk + (lo + tb) / E : nullptr;
        const size_t bstride = (size_t)P.nrows * (size_t)P.nblk;
        if (GUARD && (slowbits & P.guard_hist)) {
            for (int iw = 0; iw < P.nw; ++iw, zp += plane) {
                const int w = P.w[iw];
                const float scl = P.scale[iw];
                const int lim = nrem - w;
                float ss = 0.f, mx = -INFINITY;
#pragma unroll 1
                for (int k = 0; k < V; ++k) {
                    const int o = ob + k * NT;
                    if (o < 0 || o >= seglen) continue;
                    long long zz = 0;
                    if (o <= lim) {
                        int sl = rslot + j + k * NT;      // recomputed: no dynamic register-array index
                        if (sl >= RING) sl -= RING;
                        uint32_t prev = (uint32_t)ring[sl];
                        for (int q = 0; q < w; ++q) {
                            if (++sl >= RING) sl = 0;
                            const uint32_t cur = (uint32_t)ring[sl];
                            zz += (long long)(int)(cur - prev);
                            prev = cur;
                        }
                    }
                    const float z = (float)zz * scl;
                    if (RMS) { ss = __fmaf_rn(z, z, ss); mx = fmaxf(mx, z); }
                    __stcs(zp + k * NT, z);
                }
                if (RMS) sAcc[iw * NT + j] += ss;
                if (RMS && bmax) push_block_max(bmax + (size_t)iw * bstride, mx);
            }
        } else if (interior) {
            for (int iw = 0; iw < P.nw; ++iw, zp += plane) {
                const int w = P.w[iw];
                const float scl = P.scale[iw];
                float ss = 0.f, mx = -INFINITY;
#pragma unroll
                for (int k = 0; k < V; ++k) {
                    int sl = rs[k] + w;
                    if (!MIRROR && sl >= RING) sl -= RING;
                    const float z = acc_to_float((ACC)(ring[sl] - p0[k])) * scl;
                    if (RMS) { ss = __fmaf_rn(z, z, ss); mx = fmaxf(mx, z); }
                    __stcs(zp + k * NT, z);
                }
                if (RMS) sAcc[iw * NT + j] += ss;
                if (RMS && bmax) push_block_max(bmax + (size_t)iw * bstride, mx);
            }
        } else {
            for (int iw = 0; iw < P.nw; ++iw, zp += plane) {
                const int w = P.w[iw];
                const float scl = P.scale[iw];
                const int lim = nrem - w;                 // t + w <= n  <=>  o <= lim
                float ss = 0.f, mx = -INFINITY;
#pragma unroll
                for (int k = 0; k < V; ++k) {
                    const int o = ob + k * NT;
                    if (o >= 0 && o < seglen) {
                        int sl = rs[k] + w;
                        if (!MIRROR && sl >= RING) sl -= RING;
                        const float z = (o <= lim) ? acc_to_float((ACC)(ring[sl] - p0[k])) * scl : 0.f;
                        if (RMS) { ss = __fmaf_rn(z, z, ss); mx = fmaxf(mx, z); }
                        __stcs(zp + k * NT, z);           // streaming store: keep x, not z, in L2
                    }
                }
                if (RMS) sAcc[iw * NT + j] += ss;
                if (RMS && bmax) push_block_max(bmax + (size_t)iw * bstride, mx);
            }
        }
        wslot += E;
        if (wslot >= RING) wslot -= RING;
        rslot += E;
        if (rslot >= RING) rslot -= RING;
        __syncthreads();
    }
    if (RMS) {
        // block sum per width in float64, fixed order: lanes by shuffle, then the 8 warp sums in sequence
        double *sw = reinterpret_cast<double *>(sX);      // sX is free now: [NT/32] doubles
        for (int iw = 0; iw < P.nw; ++iw) {
            double v = (double)sAcc[iw * NT + j];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
            if ((j & 31) == 0) sw[j >> 5] = v;
            __syncthreads();
            if (j == 0) {
                double t = 0.0;
                for (int q = 0; q < NT / 32; ++q) t += sw[q];
                P.partial[((size_t)iw * (size_t)P.nrows + (size_t)row) * P.nseg + seg] = t;
            }
            __syncthreads();
        }
    }
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

namespace {
long long mf_segment(long long nsamps)
{
    // segments: about 8 steps each, so that the grid is many waves deep
    long long seg = 8ll * E;
    if (seg > nsamps) seg = (nsamps + E - 1) / E * E;
    return seg;
}
}  // namespace

// The dense pass (z written; with rms_dev also the RMS and, optionally, the block maxima) runs the CTA-cooperative
// kernel of this file.  Passes that store no dense z -- z_dev null with rms_dev given (RMS + block maxima only), and
// the sparse re-computation of listed blocks into a compact z (sparse_list / sparse_count / zc / max_blocks:
// dedisp_search_events) -- run the warp-autonomous kernel of matched_filter_warp.cu.  z is bit-identical between
// the two kernels (exact integer numerators); their RMS agrees to the documented 2^-20 (different summation order).
dedisp_status mf_run(const void *x_dev, dedisp_out_dtype x_dtype, long long nrows, long long nsamps, int radius,
                     const int *widths_host, int nwidths, unsigned int x_max, float *z_dev, float *rms_dev,
                     int *blockmax_dev, void *workspace_dev, size_t workspace_bytes, void *cuda_stream,
                     const int2 *sparse_list, const int *sparse_count, float *zc, long long max_blocks)
{
    // (A/B hook: DEDISP_MF_WARP_DENSE=1 sends the dense pass of dedisp_matched_filter_rms -- which has a workspace for
    // the prefix sums -- through the warp kernel too; profiles/r2_matched_filter.md)
    static const bool warp_dense = getenv("DEDISP_MF_WARP_DENSE") != nullptr;
    if (sparse_list || !z_dev || (warp_dense && rms_dev && workspace_dev))
        return mf_warp_run(x_dev, x_dtype, nrows, nsamps, radius, widths_host, nwidths, x_max, z_dev, rms_dev, blockmax_dev,
                           workspace_dev, workspace_bytes, cuda_stream, sparse_list, sparse_count, zc, max_blocks);
    if (!x_dev || !widths_host || nrows < 1 || nsamps < 1 || radius < 0)
        return DEDISP_ERR_INVALID_ARG;
    if (x_dtype != DEDISP_OUT_U32 && x_dtype != DEDISP_OUT_F32) return DEDISP_ERR_UNSUPPORTED_DTYPE;
    if (nwidths < 1 || nwidths > MAXW || nsamps > (1ll << 30)) return DEDISP_ERR_INVALID_ARG;
    if (((uintptr_t)x_dev & 3u) || ((uintptr_t)z_dev & 3u)) return DEDISP_ERR_INVALID_ARG;
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
    const int ring = (E + P.wmax + 1 + 7) & ~7;
    P.ring = ring;
    const long long seg = mf_segment(nsamps);
    P.seg = (int)seg;
    const long long nseg = (nsamps + seg - 1) / seg;
    P.nseg = (int)nseg;
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
    P.guard_hist = (1 << ((P.wmax + E - 1) / E + 1)) - 1;
    const size_t accb = wide ? 8 : 4;
    const bool rms = rms_dev != nullptr;
    P.partial = (double *)workspace_dev;
    P.blockmax = blockmax_dev;
    P.nblk = (int)((nsamps + P.wmax + E - 1) / E);
    if (blockmax_dev && (!rms || ((uintptr_t)blockmax_dev & 3u))) return DEDISP_ERR_INVALID_ARG;
    if (rms) {
        if (!workspace_dev || ((uintptr_t)workspace_dev & 7u) || ((uintptr_t)rms_dev & 3u) ||
            workspace_bytes < (size_t)nwidths * (size_t)nrows * (size_t)nseg * sizeof(double))
            return DEDISP_ERR_INVALID_ARG;
    }
    const size_t smem = 2 * (size_t)E * 4 + (NT / 32) * accb + (wide ? 1 : 2) * (size_t)ring * accb +
                        (rms ? (size_t)nwidths * NT * 4 : 0);
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const dim3 grid((unsigned)(nrows * nseg)), block(NT);
    cudaError_t e = cudaSuccess;
    if (blockmax_dev &&   // every byte 0x80: below the image of any finite float
        cudaMemsetAsync(blockmax_dev, 0x80, (size_t)nwidths * (size_t)nrows * (size_t)P.nblk * 4, s) != cudaSuccess)
        return DEDISP_ERR_CUDA;
#define MF_LAUNCH1(ACC, F, G, R)                                                                  \
    do {                                                                                         \
        e = cudaFuncSetAttribute(matched_filter_kernel<ACC, F, G, R>,                            \
                                 cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);        \
        if (e == cudaSuccess) matched_filter_kernel<ACC, F, G, R><<<grid, block, smem, s>>>(P);  \
    } while (0)
#define MF_LAUNCH(ACC, F, G)                     \
    do {                                         \
        if (rms) MF_LAUNCH1(ACC, F, G, true);    \
        else MF_LAUNCH1(ACC, F, G, false);       \
    } while (0)
    const bool f32 = (x_dtype == DEDISP_OUT_F32);
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
#undef MF_LAUNCH
#undef MF_LAUNCH1
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e != cudaSuccess) return DEDISP_ERR_CUDA;
    ++g_launch_count;
    if (rms) {
        const long long nseries = (long long)nwidths * nrows;
        mf_rms_finish_kernel<<<(unsigned)((nseries + 255) / 256), 256, 0, s>>>(P.partial, nseries, P.nseg, nsamps, rms_dev);
        if (cudaGetLastError() != cudaSuccess) return DEDISP_ERR_CUDA;
        ++g_launch_count;
    }
    return DEDISP_OK;
}

extern "C" dedisp_status dedisp_matched_filter(const void *x_dev, dedisp_out_dtype x_dtype,
                                               long long nrows, long long nsamps, int radius,
                                               const int *widths_host, int nwidths,
                                               unsigned int x_max, float *z_dev, void *cuda_stream)
{
    if (!z_dev) return DEDISP_ERR_INVALID_ARG;
    return mf_run(x_dev, x_dtype, nrows, nsamps, radius, widths_host, nwidths, x_max, z_dev, nullptr, nullptr, nullptr,
                  0, cuda_stream, nullptr, nullptr, nullptr, 0);
}

extern "C" size_t dedisp_matched_filter_rms_workspace_bytes(long long nrows, long long nsamps, int nwidths)
{
    if (nrows < 1 || nsamps < 1 || nwidths < 1 || nwidths > MAXW) return 0;
    const long long seg = mf_segment(nsamps);     // either kernel may serve the call
    const size_t a = (size_t)nwidths * (size_t)nrows * (size_t)((nsamps + seg - 1) / seg) * sizeof(double);
    const size_t b = mf_warp_workspace_bytes(nrows, nsamps, nwidths);
    return a > b ? a : b;
}

extern "C" dedisp_status dedisp_matched_filter_rms(const void *x_dev, dedisp_out_dtype x_dtype, long long nrows,
                                                   long long nsamps, int radius, const int *widths_host,
                                                   int nwidths, unsigned int x_max, float *z_dev, float *rms_dev,
                                                   int *blockmax_dev, void *workspace_dev, size_t workspace_bytes,
                                                   void *cuda_stream)
{
    if (!rms_dev) return DEDISP_ERR_INVALID_ARG;      // (z_dev may be null: RMS and block maxima only, z is not written)
    return mf_run(x_dev, x_dtype, nrows, nsamps, radius, widths_host, nwidths, x_max, z_dev, rms_dev, blockmax_dev,
                  workspace_dev, workspace_bytes, cuda_stream, nullptr, nullptr, nullptr, 0);
}

extern "C" long long dedisp_matched_filter_hint_blocks(long long nsamps, const int *widths_host, int nwidths,
                                                       int *hint_block, int *hint_offset)
{
    if (nsamps < 1 || !widths_host || nwidths < 1 || nwidths > MAXW) return 0;
    int wmax = 0;
    for (int i = 0; i < nwidths; ++i) {
        if (widths_host[i] < 1 || widths_host[i] > DEDISP_MF_MAX_WIDTH) return 0;
        if (widths_host[i] > wmax) wmax = widths_host[i];
    }
    if (hint_block) *hint_block = E;
    if (hint_offset) *hint_offset = wmax;
    return (nsamps + wmax + E - 1) / E;
}
