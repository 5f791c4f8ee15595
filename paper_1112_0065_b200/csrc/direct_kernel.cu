// direct_kernel.cu -- the plain gather-sum straight from the definition
//   out[d][t] = sum_c in[c][t + delay[c][d]]        (BASELINE.json:north_star)
// One thread per output sample, samples extracted from the packed rows in global
// memory.  It serves any plan (unsorted DM lists, huge DM steps, odd sizes) and is
// the fallback of DEDISP_KERNEL_AUTO when the bit-sliced kernel's tile window does
// not fit; it is also the "before" row of the ncu evidence table in DESIGN.md.
#include "dedisp_internal.h"

template <int NBITS, bool F32>
__global__ void __launch_bounds__(256)
direct_kernel(const int32_t *__restrict__ delay, int nchans, int ndm, long long nsamps_out,
              const uint8_t *__restrict__ in, size_t row_stride, size_t in_beam_stride,
              uint8_t *__restrict__ out, size_t out_beam_stride)
{
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int d = blockIdx.y;
    const int b = blockIdx.z;
    if (t >= nsamps_out) return;
    const uint8_t *inb = in + (size_t)b * in_beam_stride;
    uint32_t acc = 0;
    for (int c = 0; c < nchans; ++c) {
        const long long ti = t + __ldg(&delay[(size_t)c * ndm + d]);
        const uint8_t *row = inb + (size_t)c * row_stride;
        if (NBITS == 8) {
            acc += row[ti];
        } else {   // LSB-first sub-byte samples: bits [ti*NBITS, (ti+1)*NBITS) of the row
            const long long bit = ti * NBITS;
            acc += (row[bit >> 3] >> (int)(bit & 7)) & ((1u << NBITS) - 1u);
        }
    }
    uint8_t *ob = out + (size_t)b * out_beam_stride;
    const size_t idx = (size_t)d * (size_t)nsamps_out + (size_t)t;
    if (F32)
        reinterpret_cast<float *>(ob)[idx] = (float)acc;
    else
        reinterpret_cast<uint32_t *>(ob)[idx] = acc;
}

cudaError_t launch_direct(const int32_t *d_delay, int nchans, int ndm, long long nsamps_out,
                          const uint8_t *in, size_t row_stride, size_t in_beam_stride, int nbits,
                          void *out, size_t out_beam_stride, int out_f32, int nbeams,
                          cudaStream_t s)
{
    // grid.y/z are limited to 65535: loop over DM slabs if ever needed
    const int DSLAB = 65535;
    for (int d0 = 0; d0 < ndm; d0 += DSLAB) {
        const int nd = (ndm - d0 < DSLAB) ? (ndm - d0) : DSLAB;
        dim3 block(256), grid((unsigned)((nsamps_out + 255) / 256), nd, nbeams);
        const int32_t *dl = d_delay + d0;
        uint8_t *o = (uint8_t *)out + (size_t)d0 * (size_t)nsamps_out * 4;
#define LAUNCH(NB, F)                                                                            \
    direct_kernel<NB, F><<<grid, block, 0, s>>>(dl, nchans, ndm, nsamps_out, in, row_stride,     \
                                                in_beam_stride, o, out_beam_stride)
        if (nbits == 2 && !out_f32) LAUNCH(2, false);
        else if (nbits == 2) LAUNCH(2, true);
        else if (nbits == 1 && !out_f32) LAUNCH(1, false);
        else if (nbits == 1) LAUNCH(1, true);
        else if (nbits == 4 && !out_f32) LAUNCH(4, false);
        else if (nbits == 4) LAUNCH(4, true);
        else if (!out_f32) LAUNCH(8, false);
        else LAUNCH(8, true);
#undef LAUNCH
        ++g_launch_count;
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}
