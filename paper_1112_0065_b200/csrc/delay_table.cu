// delay_table.cu -- kernel A: device delay-table builder (north_star subsystem (a)).
//
//   delay[c][d] = round_half_away( ((4148.808*DM_d) * (1/(f_c*f_c) - 1/(f_top*f_top))) / dt )
//   f_c = f_top + c*df
//
// BASELINE.json:north_star gives the formula ("rounding is to nearest with ties away
// from zero, evaluated in double"); the paper itself only says "frequency-dependent
// time delay" (Sec. 2.2).  Every operation is an explicit IEEE
// round-to-nearest intrinsic so that nvcc cannot contract a*b+c into an FMA.
#include "dedisp_internal.h"

__global__ void delay_table_kernel(int nchans, double dt, double f_top, double df,
                                   const double *__restrict__ dms, int ndm,
                                   int32_t *__restrict__ delay, int *max_delay, int *overflow)
{
    const int d = blockIdx.x * blockDim.x + threadIdx.x;
    int v = 0;
    for (int c = blockIdx.y; c < nchans; c += gridDim.y) {
        if (d >= ndm) break;
        const double fc = __dadd_rn(f_top, __dmul_rn((double)c, df));
        const double a = __dsub_rn(__ddiv_rn(1.0, __dmul_rn(fc, fc)),
                                   __ddiv_rn(1.0, __dmul_rn(f_top, f_top)));
        const double x = __ddiv_rn(__dmul_rn(__dmul_rn(4148.808, dms[d]), a), dt);
        // nearest, ties away from zero; x - trunc(x) is exact in double
        double r = trunc(x);
        const double frac = __dsub_rn(x, r);
        if (frac >= 0.5) r = __dadd_rn(r, 1.0);
        if (frac <= -0.5) r = __dsub_rn(r, 1.0);
        if (!(r >= 0.0) || r > 2147483000.0) {
            atomicExch(overflow, 1);
            r = 0.0;
        }
        delay[(size_t)c * ndm + d] = (int)r;
        v = max(v, (int)r);
    }
    // block max -> one atomic per warp
    for (int o = 16; o > 0; o >>= 1) v = max(v, __shfl_xor_sync(0xffffffffu, v, o));
    if ((threadIdx.x & 31) == 0 && v > 0) atomicMax(max_delay, v);
}

cudaError_t launch_delay_table(int nchans, double dt, double f_top, double df, const double *d_dms,
                               int ndm, int32_t *d_delay, int *d_max_delay, int *d_overflow,
                               cudaStream_t s)
{
    dim3 block(128), grid((ndm + 127) / 128, nchans < 65535 ? nchans : 65535);
    delay_table_kernel<<<grid, block, 0, s>>>(nchans, dt, f_top, df, d_dms, ndm, d_delay,
                                              d_max_delay, d_overflow);
    ++g_launch_count;
    return cudaGetLastError();
}
