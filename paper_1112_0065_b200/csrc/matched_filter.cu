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
// word, so 32-bit words serve whenever wmax*N*x_max < 2^31 and 64-bit words otherwise.
// A work item is (row, segment of SEG samples); a CTA walks its segment in steps of
// E = NT*V samples: coalesced loads of the three input streams (x[t], x[t+R],
// x[t-R-1]; the two trailing streams hit L2), two block scans, then the outputs of
// the step that lags wmax samples behind, written with coalesced 4-byte stores.
#include <cmath>
#include <type_traits>

#include "dedisp_internal.h"

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
    int ring;                    // ring entries, power of two >= E + wmax + 1
    int seg;                     // samples per segment (multiple of E)
    int nseg;
    int w[MAXW];
    float scale[MAXW];           // fl32(1 / (N sqrt(w)))
};

__device__ __forceinline__ int pad(int i) { return i + (i >> 5); }

template <bool XF32>
__device__ __forceinline__ uint32_t load_x(const void *x, long long idx)
{
    if (XF32) return (uint32_t)__ldg(reinterpret_cast<const float *>(x) + idx);
    return __ldg(reinterpret_cast<const uint32_t *>(x) + idx);
}

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
    ACC base = 0, tot = 0;
#pragma unroll
    for (int k = 0; k < NT / 32; ++k) {
        const ACC s = sc[k];
        if (k < warp) base += s;
        tot += s;
    }
    total = tot;
    __syncthreads();
    return v + base;
}

template <class ACC, bool XF32>
__global__ void __launch_bounds__(NT) matched_filter_kernel(const MFParams P)
{
    typedef typename std::conditional<sizeof(ACC) == 8, long long, int>::type SACC;
    extern __shared__ __align__(16) uint8_t smem_raw[];
    uint32_t *sX = reinterpret_cast<uint32_t *>(smem_raw);          // [pad(E)]
    uint32_t *sD = sX + (E + E / 32);                               // [pad(E)]  x[t+R] - x[t-R-1]
    ACC *sc = reinterpret_cast<ACC *>(sD + (E + E / 32));           // [NT/32]
    ACC *ring = sc + NT / 32;                                       // [ring + ring/32]
    const int rmask = P.ring - 1;

    const long long row = blockIdx.x / P.nseg;
    const int seg = (int)(blockIdx.x % P.nseg);
    const long long n = P.n;
    const long long R = P.radius, N = 2 * R + 1;
    const long long lo = (long long)seg * P.seg;
    const long long hi = (lo + P.seg < n) ? lo + P.seg : n;
    const long long xrow = row * n;
    const int j = threadIdx.x;

    // window sum of the sample before the segment: a0 = clip(lo-1-R, 0, n-N)
    long long a0 = lo - 1 - R;
    if (a0 < 0) a0 = 0;
    if (a0 > n - N) a0 = n - N;
    ACC part = 0;
    for (long long k = j; k < N; k += NT) part += (ACC)load_x<XF32>(P.x, xrow + a0 + k);
    ACC carryW;
    block_scan<ACC>(part, sc, carryW);
    ACC carryP = 0;                         // P[lo] = 0: only differences are used
    if (j == 0) ring[pad((int)(lo & rmask))] = 0;

    for (long long h = lo; h < hi + P.wmax; h += E) {
        // ---- the three input streams, coalesced ----
#pragma unroll
        for (int k = 0; k < V; ++k) {
            const int i = j + k * NT;
            const long long t = h + i;
            uint32_t xt = 0, d = 0;
            if (t < n) {
                xt = load_x<XF32>(P.x, xrow + t);
                if (t >= R + 1 && t <= n - R - 1)
                    d = load_x<XF32>(P.x, xrow + t + R) - load_x<XF32>(P.x, xrow + t - R - 1);
            }
            sX[pad(i)] = xt;
            sD[pad(i)] = d;
        }
        __syncthreads();
        // ---- running window sum: scan of d ----
        ACC wv[V];
        ACC run = 0;
#pragma unroll
        for (int k = 0; k < V; ++k) {
            run += (ACC)(SACC)(int)sD[pad(j * V + k)];   // d is a signed difference
            wv[k] = run;
        }
        ACC tot;
        ACC inc = block_scan<ACC>(run, sc, tot);
        const ACC wbase = carryW + (inc - run);
        carryW += tot;
        // ---- NY = N*x - Wsum and its prefix sum ----
        ACC pv[V];
        run = 0;
#pragma unroll
        for (int k = 0; k < V; ++k) {
            const long long t = h + j * V + k;
            ACC ny = (ACC)N * (ACC)sX[pad(j * V + k)] - (wbase + wv[k]);
            if (t >= n) ny = 0;
            run += ny;
            pv[k] = run;
        }
        inc = block_scan<ACC>(run, sc, tot);
        const ACC pbase = carryP + (inc - run);
        carryP += tot;
#pragma unroll
        for (int k = 0; k < V; ++k)   // P[t+1]
            ring[pad((int)((h + j * V + k + 1) & rmask))] = pbase + pv[k];
        __syncthreads();
        // ---- outputs of the step that lags wmax behind ----
#pragma unroll 2
        for (int k = 0; k < V; ++k) {
            const long long t = h - P.wmax + j + k * NT;
            if (t < lo || t >= hi) continue;
            const ACC p0 = ring[pad((int)(t & rmask))];
            for (int iw = 0; iw < P.nw; ++iw) {
                const int w = P.w[iw];
                float z = 0.f;
                if (t + w <= n) {
                    const ACC dz = ring[pad((int)((t + w) & rmask))] - p0;
                    z = (float)(SACC)dz * P.scale[iw];
                }
                P.z[((size_t)iw * (size_t)P.nrows + (size_t)row) * (size_t)n + (size_t)t] = z;
            }
        }
        __syncthreads();
    }
}

}  // namespace

extern "C" dedisp_status dedisp_matched_filter(const void *x_dev, dedisp_out_dtype x_dtype,
                                               long long nrows, long long nsamps, int radius,
                                               const int *widths_host, int nwidths,
                                               unsigned int x_max, float *z_dev, void *cuda_stream)
{
    if (!x_dev || !z_dev || !widths_host || nrows < 1 || nsamps < 1 || radius < 0)
        return DEDISP_ERR_INVALID_ARG;
    if (x_dtype != DEDISP_OUT_U32 && x_dtype != DEDISP_OUT_F32) return DEDISP_ERR_UNSUPPORTED_DTYPE;
    if (nwidths < 1 || nwidths > MAXW) return DEDISP_ERR_INVALID_ARG;
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
    int ring = 1;
    while (ring < E + P.wmax + 1) ring <<= 1;
    P.ring = ring;
    // segments: about 8 steps each, so that the grid is many waves deep
    long long seg = 8ll * E;
    if (seg > nsamps) seg = (nsamps + E - 1) / E * E;
    P.seg = (int)seg;
    const long long nseg = (nsamps + seg - 1) / seg;
    P.nseg = (int)nseg;
    if (nrows * nseg > 0x7fffffffll) return DEDISP_ERR_INVALID_ARG;
    // |boxcar numerator| <= wmax * N * x_max must fit the signed accumulator
    const long double bound = (long double)P.wmax * (long double)N * (long double)x_max;
    if (bound >= 9.0e18L) return DEDISP_ERR_OVERFLOW;
    const bool wide = bound >= 2147483648.0L;
    const size_t accb = wide ? 8 : 4;
    const size_t smem = 2 * (size_t)(E + E / 32) * 4 + (NT / 32) * accb + (size_t)(ring + ring / 32 + 1) * accb;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const dim3 grid((unsigned)(nrows * nseg)), block(NT);
    cudaError_t e = cudaSuccess;
#define MF_LAUNCH(ACC, F)                                                                        \
    do {                                                                                         \
        e = cudaFuncSetAttribute(matched_filter_kernel<ACC, F>,                                  \
                                 cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);        \
        if (e == cudaSuccess) matched_filter_kernel<ACC, F><<<grid, block, smem, s>>>(P);        \
    } while (0)
    const bool f32 = (x_dtype == DEDISP_OUT_F32);
    if (wide) {
        if (f32) MF_LAUNCH(unsigned long long, true);
        else MF_LAUNCH(unsigned long long, false);
    } else {
        if (f32) MF_LAUNCH(uint32_t, true);
        else MF_LAUNCH(uint32_t, false);
    }
#undef MF_LAUNCH
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e != cudaSuccess) return DEDISP_ERR_CUDA;
    ++g_launch_count;
    return DEDISP_OK;
}
