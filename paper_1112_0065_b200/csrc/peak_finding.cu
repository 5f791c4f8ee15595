// peak_finding.cu -- sigma-cut + grouping of contiguous regions into events
// (Sec. 2.3: "first performing a sigma-cut and
// then gathering contiguous regions together into individual events ... 'transform' and
// 'reduce_by_key'"), and the per-series RMS offered as the sigma estimate.
//
//   m[s][t] = z[s][t] > nsigma * sigma[s]          (float32 product, strict >, NaN never above)
//   event   = maximal run of consecutive t of one series with m true
//           -> (series, t_start, length, t_peak = first position of the maximum, peak)
//   events listed in ascending (series, t_start) order, at most max_events of them.
//
// B200 design: z (the large array) is read ONCE, coalesced, by the transform kernel, which
// leaves a bit mask (1 bit per sample: 3 % of the bytes) and the number of run starts per
// 1024-sample chunk.  Two small scans turn the counts into output offsets, so the list
// comes out sorted and deterministic without atomics or a sort.  The grouping kernel then
// works on the bit mask only and re-reads z just inside the runs (sparse).
#include "dedisp_internal.h"

namespace {

constexpr int CHUNK_WORDS = 32;                  // one warp: 32 mask words
constexpr int CHUNK = CHUNK_WORDS * 32;          // = 1024 samples per chunk
constexpr int WARPS = 8;                         // chunks per CTA in the transform kernel

struct PFLayout {
    long long nwords;        // mask words per series (multiple of CHUNK_WORDS)
    long long nchunks;       // chunks per series
    size_t off_counts, off_chunk_off, off_series_tot, off_series_base, total;
};

PFLayout make_layout(long long nseries, long long nsamps)
{
    PFLayout L;
    L.nchunks = (nsamps + CHUNK - 1) / CHUNK;
    L.nwords = L.nchunks * CHUNK_WORDS;
    size_t o = (size_t)nseries * (size_t)L.nwords * 4;          // mask
    L.off_counts = o;
    o += (size_t)nseries * (size_t)L.nchunks * 4;
    L.off_chunk_off = o;
    o += (size_t)nseries * (size_t)L.nchunks * 4;
    L.off_series_tot = o;
    o += (size_t)nseries * 4;
    o = (o + 7) & ~(size_t)7;
    L.off_series_base = o;
    o += (size_t)nseries * 8;
    L.total = o;
    return L;
}

// Where the kernels read z.  DenseZ: the full [nseries][n] array.  CompactZ (dedisp_search_events): only the blocks of
// hblock outputs whose maximum exceeds the threshold exist, re-computed into zc[index][hblock]; map[s][b] is the index
// of block b of series s (block b holds t with b*hblock - hoff <= t < (b+1)*hblock - hoff) or -1, and a sample of a
// block that does not exist is at or below the threshold by construction: it reads as -infinity.
struct DenseZ {
    const float *z;
    long long n;
    static constexpr bool DENSE = true;
    __device__ __forceinline__ float at(long long s, long long t) const { return __ldcs(z + s * n + t); }
    __device__ __forceinline__ const float *row(long long s) const { return z + s * n; }
};
struct CompactZ {
    const float *zc;
    const int *map;
    long long nblk;
    int hblock, hoff;
    static constexpr bool DENSE = false;
    __device__ __forceinline__ float at(long long s, long long t) const
    {
        const long long u = t + hoff, b = u / hblock;
        const int idx = __ldg(map + s * nblk + b);
        return idx < 0 ? -INFINITY : __ldg(zc + (size_t)idx * hblock + (u - b * hblock));
    }
    __device__ __forceinline__ const float *row(long long) const { return nullptr; }
};

// run starts of a mask word: set bits whose predecessor (previous bit, or the top bit of the
// previous word for bit 0) is clear
__device__ __forceinline__ uint32_t run_starts(uint32_t m, uint32_t prev_word)
{
    return m & ~((m << 1) | (prev_word >> 31));
}

// ---- transform of one (series, chunk) by one warp ----
template <class ZA>
__device__ __forceinline__ void cut_chunk(const ZA za, long long n, long long nchunks, long long s,
                                          long long c, float thr, uint32_t *__restrict__ mask,
                                          uint32_t *__restrict__ counts, int vec_ok, int lane)
{
    const float *zr = za.row(s);
    const long long t0 = c * CHUNK;
    uint32_t mine = 0;
    if (!ZA::DENSE) {
        for (int w = 0; w < CHUNK_WORDS; ++w) {
            const long long t = t0 + w * 32 + lane;
            const uint32_t b = __ballot_sync(0xffffffffu, t < n && za.at(s, t) > thr);
            if (lane == w) mine = b;
        }
    } else if (vec_ok && t0 + CHUNK <= n) {
        // 128-bit loads: lane l of pass i holds samples 128 i + 4 l .. + 3 -> a nibble of word
        // 4 i + l/8; three OR-shuffles assemble the word in its 8-lane group, one more hands word
        // L to lane L
        const float4 *z4 = reinterpret_cast<const float4 *>(zr + t0);
#pragma unroll
        for (int i = 0; i < CHUNK / 128; ++i) {
            const float4 q = __ldcs(z4 + i * 32 + lane);
            uint32_t v = (q.x > thr ? 1u : 0u) | (q.y > thr ? 2u : 0u) | (q.z > thr ? 4u : 0u) |
                         (q.w > thr ? 8u : 0u);
            v <<= 4 * (lane & 7);
            v |= __shfl_xor_sync(0xffffffffu, v, 1);
            v |= __shfl_xor_sync(0xffffffffu, v, 2);
            v |= __shfl_xor_sync(0xffffffffu, v, 4);
            v = __shfl_sync(0xffffffffu, v, 8 * (lane & 3));
            if ((lane >> 2) == i) mine = v;
        }
    } else if (t0 + CHUNK <= n) {
#pragma unroll 8
        for (int w = 0; w < CHUNK_WORDS; ++w) {
            const uint32_t b = __ballot_sync(0xffffffffu, __ldcs(zr + t0 + w * 32 + lane) > thr);
            if (lane == w) mine = b;
        }
    } else {
        for (int w = 0; w < CHUNK_WORDS; ++w) {
            const long long t = t0 + w * 32 + lane;
            const uint32_t b = __ballot_sync(0xffffffffu, t < n && __ldcs(zr + t) > thr);
            if (lane == w) mine = b;
        }
    }
    // top bit of the word before: previous lane, or the sample before the chunk
    uint32_t prev = __shfl_up_sync(0xffffffffu, mine, 1);
    if (lane == 0) prev = (t0 > 0 && za.at(s, t0 - 1) > thr) ? 0x80000000u : 0u;
    int cnt = __popc(run_starts(mine, prev));
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
    mask[(s * nchunks + c) * CHUNK_WORDS + lane] = mine;
    if (lane == 0) counts[s * nchunks + c] = (uint32_t)cnt;
}

// one warp per (series, chunk)
__global__ void __launch_bounds__(WARPS * 32)
sigma_cut_kernel(const DenseZ z, long long nseries, long long n, long long nchunks,
                 const float *__restrict__ sigma, float nsigma, uint32_t *__restrict__ mask,
                 uint32_t *__restrict__ counts, int vec_ok)
{
    const long long item = (long long)blockIdx.x * WARPS + (threadIdx.x >> 5);
    if (item >= nseries * nchunks) return;
    const long long s = item / nchunks;
    cut_chunk(z, n, nchunks, s, item % nchunks, __fmul_rn(nsigma, __ldg(sigma + s)), mask, counts, vec_ok,
              threadIdx.x & 31);
}

// Hinted form: mask and counts have been zeroed; a warp looks at 32 (series, chunk) items, lane = item,
// and transforms only those the hint does not rule out.  hint[s][b] bounds (order-preserving int image of
// the float) every z[s][t] with b*hint_block - hint_offset <= t < (b+1)*hint_block - hint_offset from
// above: a chunk all of whose blocks stay at or below the threshold holds no sample above it.
template <class ZA>
__global__ void __launch_bounds__(WARPS * 32)
sigma_cut_hinted_kernel(const ZA z, long long nseries, long long n, long long nchunks,
                        const float *__restrict__ sigma, float nsigma, uint32_t *__restrict__ mask,
                        uint32_t *__restrict__ counts, int vec_ok, const int *__restrict__ hint, int hint_block,
                        int hint_offset, long long hint_nblocks)
{
    const int lane = threadIdx.x & 31;
    const long long base = ((long long)blockIdx.x * WARPS + (threadIdx.x >> 5)) * 32;
    const long long nitems = nseries * nchunks;
    if (base >= nitems) return;
    const long long item = base + lane;
    bool look = false;
    float thr = 0.f;
    if (item < nitems) {
        const long long s = item / nchunks, t0 = (item % nchunks) * CHUNK;
        thr = __fmul_rn(nsigma, __ldg(sigma + s));
        const long long tl = t0 + CHUNK - 1 < n - 1 ? t0 + CHUNK - 1 : n - 1;
        const long long b1 = (tl + hint_offset) / hint_block;
        int hi = (int)0x80000000;
        for (long long b = (t0 + hint_offset) / hint_block; b <= b1; ++b) hi = max(hi, __ldg(hint + s * hint_nblocks + b));
        const int ti = __float_as_int(thr);
        look = !(thr == thr) || hi > (ti >= 0 ? ti : ti ^ 0x7fffffff);
    }
    uint32_t todo = __ballot_sync(0xffffffffu, look);
    while (todo) {
        const int src = __ffs(todo) - 1;
        todo &= todo - 1;
        const long long it = base + src;
        cut_chunk(z, n, nchunks, it / nchunks, it % nchunks, __shfl_sync(0xffffffffu, thr, src), mask, counts, vec_ok,
                  lane);
    }
}

// ---- scan 1: one warp per series: exclusive offsets of its chunks + series total ----
__global__ void __launch_bounds__(256)
chunk_scan_kernel(const uint32_t *__restrict__ counts, long long nseries, long long nchunks,
                  uint32_t *__restrict__ chunk_off, uint32_t *__restrict__ series_tot)
{
    const int lane = threadIdx.x & 31;
    const long long s = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (s >= nseries) return;
    uint32_t carry = 0;
    for (long long c0 = 0; c0 < nchunks; c0 += 32) {
        const long long c = c0 + lane;
        const uint32_t v = c < nchunks ? counts[s * nchunks + c] : 0u;
        uint32_t inc = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t u = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += u;
        }
        if (c < nchunks) chunk_off[s * nchunks + c] = carry + inc - v;
        carry += __shfl_sync(0xffffffffu, inc, 31);
    }
    if (lane == 0) series_tot[s] = carry;
}

// ---- scan 2: one CTA: exclusive 64-bit offsets of the series + grand total; each thread owns
// a run of consecutive series, one block scan in between ----
__global__ void __launch_bounds__(1024)
series_scan_kernel(const uint32_t *__restrict__ series_tot, long long nseries,
                   unsigned long long *__restrict__ series_base, long long *__restrict__ count_out)
{
    __shared__ unsigned long long sc[32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const long long per = (nseries + 1023) / 1024;
    const long long s0 = (long long)threadIdx.x * per;
    const long long s1 = s0 + per < nseries ? s0 + per : nseries;
    unsigned long long v = 0;
    for (long long q = s0; q < s1; ++q) v += series_tot[q];
    unsigned long long inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned long long u = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += u;
    }
    if (lane == 31) sc[warp] = inc;
    __syncthreads();
    unsigned long long base = 0, tot = 0;
    for (int k = 0; k < 32; ++k) {
        if (k < warp) base += sc[k];
        tot += sc[k];
    }
    unsigned long long run = base + inc - v;
    for (long long q = s0; q < s1; ++q) {
        series_base[q] = run;
        run += series_tot[q];
    }
    if (threadIdx.x == 0) *count_out = (long long)tot;
}

// ---- reduce by key: a warp takes 32 (series, chunk) items at a time, skips those in which no
// run starts (their count is 0) and handles the others one by one, lane = mask word ----
template <class ZA>
__device__ __forceinline__ void group_chunk(const ZA za, long long n, long long nchunks,
                                            const uint32_t *__restrict__ mask,
                                            const uint32_t *__restrict__ chunk_off,
                                            const unsigned long long *__restrict__ series_base,
                                            dedisp_event *__restrict__ events, long long max_events,
                                            long long item, int lane)
{
    const long long s = item / nchunks, c = item % nchunks;
    const long long nwords = nchunks * CHUNK_WORDS;
    const uint32_t *mrow = mask + s * nwords;
    const long long wi = c * CHUNK_WORDS + lane;
    const uint32_t m = mrow[wi];
    uint32_t prev = __shfl_up_sync(0xffffffffu, m, 1);
    if (lane == 0) prev = c > 0 ? mrow[wi - 1] : 0u;
    uint32_t st = run_starts(m, prev);
    const int cnt = __popc(st);
    int inc = cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int u = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += u;
    }
    unsigned long long slot = series_base[s] + chunk_off[s * nchunks + c] + (unsigned)(inc - cnt);
    while (st) {
        const int b = __ffs(st) - 1;
        st &= st - 1;
        const long long t_start = wi * 32 + b;
        // length of the run of ones from bit b; it may continue through the next words
        const uint32_t inv = ~(m >> b);
        long long len = inv ? __ffs(inv) - 1 : 32;
        if (len >= 32 - b) {
            len = 32 - b;
            for (long long w2 = wi + 1; w2 < nwords; ++w2) {
                const uint32_t mw = mrow[w2];
                if (mw == 0xffffffffu) {
                    len += 32;
                    continue;
                }
                len += __ffs(~mw) - 1;
                break;
            }
        }
        if ((long long)slot < max_events) {
            float peak = za.at(s, t_start);
            long long tp = t_start;
            for (long long t = t_start + 1; t < t_start + len; ++t) {
                const float v = za.at(s, t);
                if (v > peak) {
                    peak = v;
                    tp = t;
                }
            }
            dedisp_event e;
            e.series = (int)s;
            e.t_start = (int)t_start;
            e.length = (int)len;
            e.t_peak = (int)tp;
            e.peak = peak;
            events[slot] = e;
        }
        ++slot;
    }
}

template <class ZA>
__global__ void __launch_bounds__(WARPS * 32)
group_events_kernel(const ZA z, long long nseries, long long n, long long nchunks,
                    const uint32_t *__restrict__ mask, const uint32_t *__restrict__ counts,
                    const uint32_t *__restrict__ chunk_off,
                    const unsigned long long *__restrict__ series_base,
                    dedisp_event *__restrict__ events, long long max_events)
{
    const int lane = threadIdx.x & 31;
    const long long nitems = nseries * nchunks;
    const long long stride = (long long)gridDim.x * WARPS * 32;
    for (long long base = ((long long)blockIdx.x * WARPS + (threadIdx.x >> 5)) * 32; base < nitems;
         base += stride) {
        const long long it = base + lane;
        uint32_t has = __ballot_sync(0xffffffffu, it < nitems && counts[it] != 0u);
        while (has) {
            const int src = __ffs(has) - 1;
            has &= has - 1;
            group_chunk(z, n, nchunks, mask, chunk_off, series_base, events, max_events, base + src, lane);
        }
    }
}

// ---- sigma estimate: sqrt(mean z^2) per series, float64 accumulation in a fixed order ----
__global__ void __launch_bounds__(256)
series_rms_kernel(const float *__restrict__ z, long long n, float *__restrict__ rms)
{
    __shared__ double sc[8];
    const float *zr = z + (long long)blockIdx.x * n;
    double acc = 0.0;
    const bool vec = (((uintptr_t)zr & 15u) == 0);
    const long long nv = vec ? (n >> 2) : 0;
    const float4 *z4 = reinterpret_cast<const float4 *>(zr);
    for (long long i = threadIdx.x; i < nv; i += 256) {
        const float4 q = __ldcs(z4 + i);
        acc += (double)q.x * (double)q.x + (double)q.y * (double)q.y + (double)q.z * (double)q.z +
               (double)q.w * (double)q.w;
    }
    for (long long i = 4 * nv + threadIdx.x; i < n; i += 256) {
        const double v = (double)__ldcs(zr + i);
        acc += v * v;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) sc[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int k = 0; k < 8; ++k) t += sc[k];
        rms[blockIdx.x] = (float)sqrt(t / (double)n);
    }
}

bool pf_sizes_ok(long long nseries, long long nsamps)
{
    if (nseries < 1 || nsamps < 1 || nsamps > (1ll << 30) || nseries > 0x7fffffffll) return false;
    const long long nchunks = (nsamps + CHUNK - 1) / CHUNK;
    return nseries * nchunks <= 0x7fffffffll * (long long)WARPS / 2;
}

}  // namespace

extern "C" {

size_t dedisp_find_events_workspace_bytes(long long nseries, long long nsamps)
{
    if (!pf_sizes_ok(nseries, nsamps)) return 0;
    return make_layout(nseries, nsamps).total;
}

}  // extern "C"

// The four kernels of the event search over the z the accessor ZA presents (dense array, or compact blocks).
template <class ZA>
static dedisp_status find_events_launch(const ZA za, bool vec_ok, long long nseries, long long nsamps,
                                        const float *sigma_dev, float nsigma, const int *hint_dev, int hint_block,
                                        int hint_offset, void *workspace_dev, size_t workspace_bytes,
                                        dedisp_event *events_dev, long long max_events, long long *count_dev,
                                        cudaStream_t s)
{
    const PFLayout L = make_layout(nseries, nsamps);
    if (workspace_bytes < L.total) return DEDISP_ERR_INVALID_ARG;
    uint8_t *ws = (uint8_t *)workspace_dev;
    uint32_t *mask = (uint32_t *)ws;
    uint32_t *counts = (uint32_t *)(ws + L.off_counts);
    uint32_t *chunk_off = (uint32_t *)(ws + L.off_chunk_off);
    uint32_t *series_tot = (uint32_t *)(ws + L.off_series_tot);
    unsigned long long *series_base = (unsigned long long *)(ws + L.off_series_base);
    const long long items = nseries * L.nchunks;
    const unsigned grid = (unsigned)((items + WARPS - 1) / WARPS);
    if (hint_dev) {
        // mask and counts (adjacent in the workspace) start at zero; only the chunks the hint cannot rule out
        // are transformed
        if (cudaMemsetAsync(mask, 0, L.off_chunk_off, s) != cudaSuccess) return DEDISP_ERR_CUDA;
        const unsigned hgrid = (unsigned)((items + 32 * WARPS - 1) / (32 * WARPS));
        sigma_cut_hinted_kernel<ZA><<<hgrid, WARPS * 32, 0, s>>>(za, nseries, nsamps, L.nchunks, sigma_dev, nsigma,
                                                                 mask, counts, vec_ok, hint_dev, hint_block, hint_offset,
                                                                 (nsamps + hint_offset + hint_block - 1) / hint_block);
    } else {
        if constexpr (ZA::DENSE)
            sigma_cut_kernel<<<grid, WARPS * 32, 0, s>>>(za, nseries, nsamps, L.nchunks, sigma_dev, nsigma, mask, counts,
                                                         vec_ok);
        else
            return DEDISP_ERR_INVALID_ARG;
    }
    chunk_scan_kernel<<<(unsigned)((nseries + 7) / 8), 256, 0, s>>>(counts, nseries, L.nchunks,
                                                                    chunk_off, series_tot);
    series_scan_kernel<<<1, 1024, 0, s>>>(series_tot, nseries, series_base, count_dev);
    int sms = 148, dev = 0;
    if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const long long gwant = (items + WARPS * 32 - 1) / (WARPS * 32);
    const unsigned ggrid = (unsigned)(gwant < 8ll * sms ? gwant : 8ll * sms);
    group_events_kernel<ZA><<<ggrid, WARPS * 32, 0, s>>>(za, nseries, nsamps, L.nchunks, mask, counts,
                                                         chunk_off, series_base, events_dev, max_events);
    g_launch_count += 4;
    return cudaGetLastError() == cudaSuccess ? DEDISP_OK : DEDISP_ERR_CUDA;
}

static dedisp_status find_events_run(const float *z_dev, long long nseries, long long nsamps,
                                     const float *sigma_dev, float nsigma, const int *hint_dev, int hint_block,
                                     int hint_offset, void *workspace_dev, size_t workspace_bytes,
                                     dedisp_event *events_dev, long long max_events, long long *count_dev,
                                     void *cuda_stream)
{
    if (!z_dev || !sigma_dev || !workspace_dev || !count_dev || max_events < 0 ||
        (max_events > 0 && !events_dev))
        return DEDISP_ERR_INVALID_ARG;
    if (!pf_sizes_ok(nseries, nsamps)) return DEDISP_ERR_INVALID_ARG;
    if (((uintptr_t)z_dev & 3u) || ((uintptr_t)workspace_dev & 7u) || ((uintptr_t)events_dev & 3u) ||
        ((uintptr_t)count_dev & 7u))
        return DEDISP_ERR_INVALID_ARG;
    const bool vec_ok = (((uintptr_t)z_dev & 15u) == 0) && (nsamps % 4 == 0);
    return find_events_launch(DenseZ{z_dev, nsamps}, vec_ok, nseries, nsamps, sigma_dev, nsigma, hint_dev, hint_block,
                              hint_offset, workspace_dev, workspace_bytes, events_dev, max_events, count_dev,
                              (cudaStream_t)cuda_stream);
}

// ---- dedisp_search_events: rows f1 + f2 without materialising z ----
// One thread per (series, block): blocks whose maximum exceeds the series' threshold get a slot in the compact z
// (first come first served: the slot order is irrelevant, the event list is ordered by the scans) and are listed for
// the sparse re-computation; count[0] = number of such blocks (all of them, also beyond the capacity).
__global__ void __launch_bounds__(256)
flag_blocks_kernel(const int *__restrict__ blockmax, const float *__restrict__ sigma, float nsigma, long long nseries,
                   long long nblk, int max_blocks, int *__restrict__ map, int2 *__restrict__ list, int *count)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nseries * nblk) return;
    const long long s = i / nblk;
    const float thr = __fmul_rn(nsigma, __ldg(sigma + s));
    const int ti = __float_as_int(thr);
    const bool look = !(thr == thr) || blockmax[i] > (ti >= 0 ? ti : ti ^ 0x7fffffff);
    int slot = -1;
    if (look) {
        slot = atomicAdd(count, 1);
        if (slot < max_blocks) list[slot] = make_int2((int)s, (int)(i - s * nblk));
        else slot = -1;
    }
    map[i] = slot;
}

// count_out[1] = blocks flagged; count[0] (the sparse kernel's CTA count) = min(flagged, max_blocks)
__global__ void clamp_block_count_kernel(int *count, int max_blocks, long long *count_out)
{
    count_out[1] = *count;
    if (*count > max_blocks) *count = max_blocks;
}

struct SearchLayout {
    size_t off_partial, off_blockmax, off_map, off_list, off_count, off_zc, off_pf, total;
    long long nblk;
    int hblock, hoff;
};

static bool search_layout(long long nrows, long long nsamps, const int *widths_host, int nwidths, long long max_blocks,
                          SearchLayout &L)
{
    if (nrows < 1 || nsamps < 1 || nwidths < 1 || max_blocks < 1 || max_blocks > 0x7fffffffll) return false;
    const long long nseries = nrows * nwidths;
    if (!pf_sizes_ok(nseries, nsamps)) return false;
    L.nblk = dedisp_matched_filter_hint_blocks(nsamps, widths_host, nwidths, &L.hblock, &L.hoff);
    if (L.nblk < 1) return false;
    auto up = [](size_t v) { return (v + 255) & ~(size_t)255; };
    size_t o = 0;
    L.off_partial = o;  o = up(o + dedisp_matched_filter_rms_workspace_bytes(nrows, nsamps, nwidths));
    L.off_blockmax = o; o = up(o + (size_t)nseries * L.nblk * 4);
    L.off_map = o;      o = up(o + (size_t)nseries * L.nblk * 4);
    L.off_list = o;     o = up(o + (size_t)max_blocks * 8);
    L.off_count = o;    o = up(o + 8);
    L.off_zc = o;       o = up(o + (size_t)max_blocks * L.hblock * 4);
    L.off_pf = o;       o = up(o + dedisp_find_events_workspace_bytes(nseries, nsamps));
    L.total = o;
    return true;
}

extern "C" {

size_t dedisp_search_events_workspace_bytes(long long nrows, long long nsamps, const int *widths_host, int nwidths,
                                            long long max_blocks)
{
    SearchLayout L;
    return (widths_host && search_layout(nrows, nsamps, widths_host, nwidths, max_blocks, L)) ? L.total : 0;
}

dedisp_status dedisp_search_events(const void *x_dev, dedisp_out_dtype x_dtype, long long nrows, long long nsamps,
                                   int radius, const int *widths_host, int nwidths, unsigned int x_max, float nsigma,
                                   float *rms_dev, long long max_blocks, void *workspace_dev, size_t workspace_bytes,
                                   dedisp_event *events_dev, long long max_events, long long *count_dev,
                                   void *cuda_stream)
{
    if (!x_dev || !widths_host || !rms_dev || !workspace_dev || !count_dev || max_events < 0 ||
        (max_events > 0 && !events_dev))
        return DEDISP_ERR_INVALID_ARG;
    if (((uintptr_t)workspace_dev & 255u) || ((uintptr_t)events_dev & 3u) || ((uintptr_t)count_dev & 7u))
        return DEDISP_ERR_INVALID_ARG;
    SearchLayout L;
    if (!search_layout(nrows, nsamps, widths_host, nwidths, max_blocks, L) || workspace_bytes < L.total)
        return DEDISP_ERR_INVALID_ARG;
    uint8_t *ws = (uint8_t *)workspace_dev;
    int *blockmax = (int *)(ws + L.off_blockmax), *map = (int *)(ws + L.off_map), *count = (int *)(ws + L.off_count);
    int2 *list = (int2 *)(ws + L.off_list);
    float *zc = (float *)(ws + L.off_zc);
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const long long nseries = nrows * nwidths;
    // pass 1: the RMS of every filtered series and the block maxima of z; z itself is not written
    dedisp_status st = mf_run(x_dev, x_dtype, nrows, nsamps, radius, widths_host, nwidths, x_max, nullptr, rms_dev,
                              blockmax, ws + L.off_partial, L.off_blockmax - L.off_partial, cuda_stream, nullptr, nullptr,
                              nullptr, 0);
    if (st != DEDISP_OK) return st;
    // pass 2: the few blocks that can hold a sample above the threshold, re-computed (bit-identical: same kernel,
    // same exact integer sums) into the compact z
    if (cudaMemsetAsync(count, 0, 8, s) != cudaSuccess) return DEDISP_ERR_CUDA;
    const long long nb = nseries * L.nblk;
    flag_blocks_kernel<<<(unsigned)((nb + 255) / 256), 256, 0, s>>>(blockmax, rms_dev, nsigma, nseries, L.nblk,
                                                                    (int)max_blocks, map, list, count);
    clamp_block_count_kernel<<<1, 1, 0, s>>>(count, (int)max_blocks, count_dev);
    g_launch_count += 2;
    if (cudaGetLastError() != cudaSuccess) return DEDISP_ERR_CUDA;
    st = mf_run(x_dev, x_dtype, nrows, nsamps, radius, widths_host, nwidths, x_max, nullptr, nullptr, nullptr,
                ws + L.off_partial, L.off_blockmax - L.off_partial,      // (the prefix sums of x pass 1 left there)
                cuda_stream, list, count, zc, max_blocks);
    if (st != DEDISP_OK) return st;
    // pass 3: sigma-cut and grouping over the compact z (chunks the block maxima rule out are skipped as before)
    const CompactZ za{zc, map, L.nblk, L.hblock, L.hoff};
    return find_events_launch(za, false, nseries, nsamps, rms_dev, nsigma, blockmax, L.hblock, L.hoff, ws + L.off_pf,
                              L.total - L.off_pf, events_dev, max_events, count_dev, s);
}

dedisp_status dedisp_find_events(const float *z_dev, long long nseries, long long nsamps,
                                 const float *sigma_dev, float nsigma, void *workspace_dev,
                                 size_t workspace_bytes, dedisp_event *events_dev,
                                 long long max_events, long long *count_dev, void *cuda_stream)
{
    return find_events_run(z_dev, nseries, nsamps, sigma_dev, nsigma, nullptr, 0, 0, workspace_dev, workspace_bytes,
                           events_dev, max_events, count_dev, cuda_stream);
}

dedisp_status dedisp_find_events_hinted(const float *z_dev, long long nseries, long long nsamps,
                                        const float *sigma_dev, float nsigma, const int *hint_dev,
                                        int hint_block, int hint_offset, void *workspace_dev,
                                        size_t workspace_bytes, dedisp_event *events_dev,
                                        long long max_events, long long *count_dev, void *cuda_stream)
{
    if (!hint_dev || hint_block < 1 || hint_offset < 0 || ((uintptr_t)hint_dev & 3u)) return DEDISP_ERR_INVALID_ARG;
    return find_events_run(z_dev, nseries, nsamps, sigma_dev, nsigma, hint_dev, hint_block, hint_offset,
                           workspace_dev, workspace_bytes, events_dev, max_events, count_dev, cuda_stream);
}

dedisp_status dedisp_series_rms(const float *z_dev, long long nseries, long long nsamps,
                                float *rms_dev, void *cuda_stream)
{
    if (!z_dev || !rms_dev || nseries < 1 || nsamps < 1 || nseries > 0x7fffffffll)
        return DEDISP_ERR_INVALID_ARG;
    if (((uintptr_t)z_dev & 3u) || ((uintptr_t)rms_dev & 3u)) return DEDISP_ERR_INVALID_ARG;
    series_rms_kernel<<<(unsigned)nseries, 256, 0, (cudaStream_t)cuda_stream>>>(z_dev, nsamps, rms_dev);
    ++g_launch_count;
    return cudaGetLastError() == cudaSuccess ? DEDISP_OK : DEDISP_ERR_CUDA;
}

}  // extern "C"
