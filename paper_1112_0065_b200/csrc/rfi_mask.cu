// rfi_mask.cu -- multibeam coincidence RFI mask (PAPER.md:38-40,
// Sec. 2.1: "a signal exceeding 3 sigma in 4 or more beams ... a transform of the multibeam time
// series, where for each sample the 13 beams are checked against the thresholds and the result
// is written as a boolean RFI mask").
//
//   above[b][s][t] = x[b][s][t] > fl32( mean[b][s] + fl32( nsigma * sigma[b][s] ) )
//   mask[s][t]     = ( #beams above ) >= min_beams                      (uint8, 1 or 0)
//
// An elementwise transform, HBM-bound: 4*nbeams bytes read and 1 byte written per sample.
// A thread owns 4 consecutive samples of one series (128-bit loads per beam, one 32-bit
// store); the nbeams thresholds of the series are CTA-uniform.
#include "dedisp_internal.h"

namespace {

template <bool XF32>
__device__ __forceinline__ float to_f(uint32_t raw)
{
    return XF32 ? __uint_as_float(raw) : (float)raw;      // uint32 sums < 2^24 convert exactly
}

// COUNTS: write the number of beams above threshold (uint8) instead of the thresholded mask -- the per-GPU half of
// the coincidence test when the beams live on several GPUs (one beam per GPU is the paper's deployment,
// PAPER.md:64): the counts are summed across ranks (an all-reduce of nseries * n bytes) and thresholded by
// counts_to_mask_kernel.
template <bool XF32, bool VEC, bool COUNTS>
__global__ void __launch_bounds__(256)
rfi_mask_kernel(const uint8_t *__restrict__ x, int nbeams, long long nseries, long long n,
                size_t beam_stride, const float *__restrict__ mean, const float *__restrict__ sigma,
                float nsigma, int min_beams, uint8_t *__restrict__ mask)
{
    const long long s = blockIdx.y;
    const long long t = ((long long)blockIdx.x * 256 + threadIdx.x) * 4;
    if (t >= n) return;
    int cnt[4] = {0, 0, 0, 0};
    for (int b = 0; b < nbeams; ++b) {
        const float thr = __fadd_rn(__ldg(mean + b * nseries + s), __fmul_rn(nsigma, __ldg(sigma + b * nseries + s)));
        const uint32_t *row = reinterpret_cast<const uint32_t *>(x + (size_t)b * beam_stride) + s * n;
        if (VEC) {
            const uint4 q = __ldcs(reinterpret_cast<const uint4 *>(row + t));
            cnt[0] += to_f<XF32>(q.x) > thr;
            cnt[1] += to_f<XF32>(q.y) > thr;
            cnt[2] += to_f<XF32>(q.z) > thr;
            cnt[3] += to_f<XF32>(q.w) > thr;
        } else {
#pragma unroll
            for (int k = 0; k < 4; ++k)
                if (t + k < n) cnt[k] += to_f<XF32>(__ldcs(row + t + k)) > thr;
        }
    }
    uint8_t *m = mask + s * n + t;
    uint32_t v[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) v[k] = COUNTS ? (uint32_t)cnt[k] : (cnt[k] >= min_beams ? 1u : 0u);
    if (VEC) {
        *reinterpret_cast<uint32_t *>(m) = v[0] | (v[1] << 8) | (v[2] << 16) | (v[3] << 24);
    } else {
#pragma unroll
        for (int k = 0; k < 4; ++k)
            if (t + k < n) m[k] = (uint8_t)v[k];
    }
}

// mask[i] = counts[i] >= min_beams over a flat array (16 bytes per thread where aligned)
__global__ void __launch_bounds__(256)
counts_to_mask_kernel(const uint8_t *__restrict__ counts, long long total, int min_beams, uint8_t *__restrict__ mask,
                      int vec)
{
    const long long i = ((long long)blockIdx.x * 256 + threadIdx.x) * 16;
    if (i >= total) return;
    if (vec && i + 16 <= total) {
        const uint4 q = __ldcs(reinterpret_cast<const uint4 *>(counts + i));
        const uint32_t w[4] = {q.x, q.y, q.z, q.w};
        uint32_t o[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            o[k] = 0;
#pragma unroll
            for (int b = 0; b < 4; ++b) o[k] |= ((int)((w[k] >> (8 * b)) & 0xffu) >= min_beams ? 1u : 0u) << (8 * b);
        }
        *reinterpret_cast<uint4 *>(mask + i) = make_uint4(o[0], o[1], o[2], o[3]);
    } else {
        for (long long k = i; k < i + 16 && k < total; ++k) mask[k] = (int)counts[k] >= min_beams ? 1 : 0;
    }
}

// An event whose peak sample is masked is vetoed: its series index s becomes -1 - s (in place; order kept);
// *kept_out = number of events left un-vetoed.
__global__ void __launch_bounds__(256)
veto_events_kernel(dedisp_event *__restrict__ events, const long long *__restrict__ count, long long max_events,
                   const uint8_t *__restrict__ mask, long long nsamps, long long *kept_out)
{
    long long n = *count;
    if (n > max_events) n = max_events;
    int kept = 0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        dedisp_event e = events[i];
        if (e.series < 0) continue;                    // vetoed by an earlier call
        if (e.t_peak >= 0 && e.t_peak < nsamps && mask[e.t_peak]) events[i].series = -1 - e.series;
        else ++kept;
    }
    kept = __reduce_add_sync(0xffffffffu, kept);
    if ((threadIdx.x & 31) == 0 && kept) atomicAdd((unsigned long long *)kept_out, (unsigned long long)kept);
}

}  // namespace

static dedisp_status rfi_run(const void *x_dev, dedisp_out_dtype x_dtype, int nbeams,
                             long long nseries, long long nsamps, size_t beam_stride_bytes,
                             const float *mean_dev, const float *sigma_dev, float nsigma,
                             int min_beams, unsigned char *mask_dev, void *cuda_stream, bool counts)
{
    if (!x_dev || !mean_dev || !sigma_dev || !mask_dev || nbeams < 1 || nseries < 1 || nsamps < 1)
        return DEDISP_ERR_INVALID_ARG;
    if (counts && nbeams > 255) return DEDISP_ERR_INVALID_ARG;
    if (x_dtype != DEDISP_OUT_U32 && x_dtype != DEDISP_OUT_F32) return DEDISP_ERR_UNSUPPORTED_DTYPE;
    if (((uintptr_t)x_dev & 3u) || (beam_stride_bytes & 3u) || nseries > 65535) return DEDISP_ERR_INVALID_ARG;
    if (nbeams > 1 && beam_stride_bytes < (size_t)nseries * (size_t)nsamps * 4) return DEDISP_ERR_INVALID_ARG;
    const long long gx = (nsamps + 1023) / 1024;
    if (gx > 0x7fffffffll) return DEDISP_ERR_INVALID_ARG;
    const bool vec = (((uintptr_t)x_dev & 15u) == 0) && (beam_stride_bytes % 16 == 0) && (nsamps % 4 == 0) &&
                     (((uintptr_t)mask_dev & 3u) == 0);
    const dim3 grid((unsigned)gx, (unsigned)nseries), block(256);
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const uint8_t *x = (const uint8_t *)x_dev;
#define RFI_LAUNCH1(F, V, C)                                                                                 \
    rfi_mask_kernel<F, V, C><<<grid, block, 0, s>>>(x, nbeams, nseries, nsamps, beam_stride_bytes, mean_dev, \
                                                    sigma_dev, nsigma, min_beams, mask_dev)
#define RFI_LAUNCH(F, V)                  \
    do {                                  \
        if (counts) RFI_LAUNCH1(F, V, true); \
        else RFI_LAUNCH1(F, V, false);    \
    } while (0)
    const bool f32 = x_dtype == DEDISP_OUT_F32;
    if (f32 && vec) RFI_LAUNCH(true, true);
    else if (f32) RFI_LAUNCH(true, false);
    else if (vec) RFI_LAUNCH(false, true);
    else RFI_LAUNCH(false, false);
#undef RFI_LAUNCH
#undef RFI_LAUNCH1
    ++g_launch_count;
    return cudaGetLastError() == cudaSuccess ? DEDISP_OK : DEDISP_ERR_CUDA;
}

extern "C" dedisp_status dedisp_rfi_mask(const void *x_dev, dedisp_out_dtype x_dtype, int nbeams,
                                         long long nseries, long long nsamps, size_t beam_stride_bytes,
                                         const float *mean_dev, const float *sigma_dev, float nsigma,
                                         int min_beams, unsigned char *mask_dev, void *cuda_stream)
{
    return rfi_run(x_dev, x_dtype, nbeams, nseries, nsamps, beam_stride_bytes, mean_dev, sigma_dev, nsigma, min_beams,
                   mask_dev, cuda_stream, false);
}

extern "C" dedisp_status dedisp_rfi_beam_counts(const void *x_dev, dedisp_out_dtype x_dtype, int nbeams,
                                                long long nseries, long long nsamps, size_t beam_stride_bytes,
                                                const float *mean_dev, const float *sigma_dev, float nsigma,
                                                unsigned char *counts_dev, void *cuda_stream)
{
    return rfi_run(x_dev, x_dtype, nbeams, nseries, nsamps, beam_stride_bytes, mean_dev, sigma_dev, nsigma, 0,
                   counts_dev, cuda_stream, true);
}

extern "C" dedisp_status dedisp_rfi_mask_from_counts(const unsigned char *counts_dev, long long nseries,
                                                     long long nsamps, int min_beams, unsigned char *mask_dev,
                                                     void *cuda_stream)
{
    if (!counts_dev || !mask_dev || nseries < 1 || nsamps < 1) return DEDISP_ERR_INVALID_ARG;
    const long long total = nseries * nsamps;
    const long long blocks = (total + 4095) / 4096;
    if (blocks > 0x7fffffffll) return DEDISP_ERR_INVALID_ARG;
    const int vec = (((uintptr_t)counts_dev | (uintptr_t)mask_dev) & 15u) == 0;
    counts_to_mask_kernel<<<(unsigned)blocks, 256, 0, (cudaStream_t)cuda_stream>>>(counts_dev, total, min_beams, mask_dev,
                                                                                   vec);
    ++g_launch_count;
    return cudaGetLastError() == cudaSuccess ? DEDISP_OK : DEDISP_ERR_CUDA;
}

extern "C" dedisp_status dedisp_veto_events(dedisp_event *events_dev, const long long *count_dev, long long max_events,
                                            const unsigned char *mask_dev, long long nsamps, long long *kept_dev,
                                            void *cuda_stream)
{
    if (!count_dev || !mask_dev || !kept_dev || max_events < 0 || nsamps < 1 || (max_events > 0 && !events_dev))
        return DEDISP_ERR_INVALID_ARG;
    if (((uintptr_t)events_dev & 3u) || ((uintptr_t)count_dev & 7u) || ((uintptr_t)kept_dev & 7u))
        return DEDISP_ERR_INVALID_ARG;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    if (cudaMemsetAsync(kept_dev, 0, 8, s) != cudaSuccess) return DEDISP_ERR_CUDA;
    const long long want = (max_events + 255) / 256;
    const unsigned grid = (unsigned)(want < 1 ? 1 : want > 1184 ? 1184 : want);
    veto_events_kernel<<<grid, 256, 0, s>>>(events_dev, count_dev, max_events, mask_dev, nsamps, kept_dev);
    ++g_launch_count;
    return cudaGetLastError() == cudaSuccess ? DEDISP_OK : DEDISP_ERR_CUDA;
}
