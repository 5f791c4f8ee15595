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

template <bool XF32, bool VEC>
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
    if (VEC) {
        *reinterpret_cast<uint32_t *>(m) = (cnt[0] >= min_beams ? 1u : 0u) | (cnt[1] >= min_beams ? 0x100u : 0u) |
                                           (cnt[2] >= min_beams ? 0x10000u : 0u) |
                                           (cnt[3] >= min_beams ? 0x1000000u : 0u);
    } else {
#pragma unroll
        for (int k = 0; k < 4; ++k)
            if (t + k < n) m[k] = cnt[k] >= min_beams ? 1 : 0;
    }
}

}  // namespace

extern "C" dedisp_status dedisp_rfi_mask(const void *x_dev, dedisp_out_dtype x_dtype, int nbeams,
                                         long long nseries, long long nsamps, size_t beam_stride_bytes,
                                         const float *mean_dev, const float *sigma_dev, float nsigma,
                                         int min_beams, unsigned char *mask_dev, void *cuda_stream)
{
    if (!x_dev || !mean_dev || !sigma_dev || !mask_dev || nbeams < 1 || nseries < 1 || nsamps < 1)
        return DEDISP_ERR_INVALID_ARG;
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
#define RFI_LAUNCH(F, V)                                                                              \
    rfi_mask_kernel<F, V><<<grid, block, 0, s>>>(x, nbeams, nseries, nsamps, beam_stride_bytes, mean_dev, \
                                                 sigma_dev, nsigma, min_beams, mask_dev)
    const bool f32 = x_dtype == DEDISP_OUT_F32;
    if (f32 && vec) RFI_LAUNCH(true, true);
    else if (f32) RFI_LAUNCH(true, false);
    else if (vec) RFI_LAUNCH(false, true);
    else RFI_LAUNCH(false, false);
#undef RFI_LAUNCH
    ++g_launch_count;
    return cudaGetLastError() == cudaSuccess ? DEDISP_OK : DEDISP_ERR_CUDA;
}
