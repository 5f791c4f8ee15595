// bitslice_prepare.cu -- set-up kernels of the tiled path:
//   * tile tables (window start per (DM group, channel); per-lane offset/shift words)
//     derived ON THE DEVICE from the device delay table (north_star subsystem (a));
//   * the unpack pre-pass (north_star subsystem (b)): packed 2-bit rows -> bit planes,
//     read with 128-bit loads whatever the row alignment, de-interleaved in registers.
#include <algorithm>
#include <numeric>

#include "bitslice_common.cuh"
#include "dedisp_internal.h"

// One block per DM group g (32 sorted trial DMs = 32 lanes), threads over channels.
//   ws[g][c]        = (delay[c][lane 0] >> 5) rounded down to a multiple of 4 words
//   rel[g][c][lane] = (((delay[c][d_lane] >> 5) - ws) * 4) << 16 | (delay[c][d_lane] & 31)
// Padding lanes repeat the group's last real DM; padding channels get zeros.
__global__ void bitslice_tables_kernel(const int32_t *__restrict__ delay, int nchans, int ndm,
                                       const int32_t *__restrict__ sorted,  // [ngroups*32], -1 = pad
                                       int nchans_pad, int32_t *__restrict__ ws,
                                       uint32_t *__restrict__ rel, int *max_off_words)
{
    const int g = blockIdx.x;
    int worst = 0;
    for (int c = threadIdx.x; c < nchans_pad; c += blockDim.x) {
        const size_t row = (size_t)g * nchans_pad + c;
        if (c >= nchans) {
            ws[row] = 0;
            for (int l = 0; l < 32; ++l) rel[row * 32 + l] = 0;
            continue;
        }
        const int32_t *dl = delay + (size_t)c * ndm;
        const int d0 = sorted[g * 32];
        const int w0 = (dl[d0] >> 5) & ~3;
        ws[row] = w0;
        int last = d0;
        for (int l = 0; l < 32; ++l) {
            const int d = sorted[g * 32 + l];
            if (d >= 0) last = d;
            const int dv = dl[last];
            const int off = (dv >> 5) - w0;   // >= 0 because the list is sorted ascending
            worst = max(worst, off);
            rel[row * 32 + l] = ((uint32_t)(off * 4) << 16) | (uint32_t)(dv & 31);
        }
    }
    for (int o = 16; o > 0; o >>= 1) worst = max(worst, __shfl_xor_sync(0xffffffffu, worst, o));
    if ((threadIdx.x & 31) == 0) atomicMax(max_off_words, worst);
}

// ---- unpack pre-pass -------------------------------------------------------
// The aligned 16-byte block at a0, restricted to the caller's buffer [vb, ve): one 128-bit load when the block lies
// inside it, byte loads of the bytes inside it otherwise (only the partial first / last block of the whole buffer
// takes that path), zero when it lies outside.  Nothing outside the caller's buffer is ever read.
__device__ __forceinline__ uint4 load_block16(uintptr_t a0, const uint8_t *vb, const uint8_t *ve)
{
    if (a0 >= (uintptr_t)vb && a0 + 16 <= (uintptr_t)ve) return __ldg(reinterpret_cast<const uint4 *>(a0));
    uint32_t w[4] = {0u, 0u, 0u, 0u};
    if (a0 + 16 > (uintptr_t)vb && a0 < (uintptr_t)ve) {
        for (int k = 0; k < 16; ++k) {
            const uintptr_t a = a0 + k;
            if (a >= (uintptr_t)vb && a < (uintptr_t)ve)
                w[k >> 2] |= (uint32_t)__ldg(reinterpret_cast<const uint8_t *>(a)) << (8 * (k & 3));
        }
    }
    return make_uint4(w[0], w[1], w[2], w[3]);
}
__device__ __forceinline__ uint32_t even_bits_to_low16(uint32_t x)
{
    x &= 0x55555555u;
    x = (x | (x >> 1)) & 0x33333333u;
    x = (x | (x >> 2)) & 0x0f0f0f0fu;
    x = (x | (x >> 4)) & 0x00ff00ffu;
    x = (x | (x >> 8)) & 0x0000ffffu;
    return x;
}

// Thread i of a row turns input bytes [16i, 16i+16) (64 two-bit samples) into two
// words of plane 0 and two words of plane 1.  The two aligned 16-byte vectors that
// cover those bytes are loaded with 128-bit loads and byte-aligned in registers.
__global__ void __launch_bounds__(128)
planes2_kernel(const uint8_t *__restrict__ in, size_t in_beam_stride, size_t row_stride,
               int nchans, const uint8_t *valid_begin, const uint8_t *valid_end,
               uint32_t *__restrict__ planes, int row_pitch, int nchans_pad)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;   // 64-sample block
    const int c = blockIdx.y, b = blockIdx.z;
    if (2 * i >= row_pitch) return;
    uint32_t r[4] = {0u, 0u, 0u, 0u};
    const long long nvalid = (long long)row_stride - 16ll * i;   // bytes of this row still valid
    if (c < nchans && nvalid > 0) {
        const uint8_t *a = in + (size_t)b * in_beam_stride + (size_t)c * row_stride + 16u * (size_t)i;
        const uintptr_t a0 = (uintptr_t)a & ~(uintptr_t)15;
        const int m = (int)((uintptr_t)a & 15);
        const uint4 lo = load_block16(a0, valid_begin, valid_end);
        const uint4 hi = m ? load_block16(a0 + 16, valid_begin, valid_end) : make_uint4(0, 0, 0, 0);
        const uint32_t v[8] = {lo.x, lo.y, lo.z, lo.w, hi.x, hi.y, hi.z, hi.w};
        const int q = m >> 2, sh = (m & 3) * 8;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            uint32_t x0 = v[k], x1 = v[k + 1];
            if (q == 1) { x0 = v[k + 1]; x1 = v[k + 2]; }
            if (q == 2) { x0 = v[k + 2]; x1 = v[k + 3]; }
            if (q == 3) { x0 = v[k + 3]; x1 = v[k + 4 < 8 ? k + 4 : 7]; }
            r[k] = __funnelshift_r(x0, x1, sh);
            // zero the bytes past the end of the row
            const long long nb = nvalid - 4 * k;
            if (nb <= 0) r[k] = 0;
            else if (nb < 4) r[k] &= (1u << (8 * (int)nb)) - 1u;
        }
    }
    if (c < nchans_pad) {
        uint2 p0, p1;
        p0.x = even_bits_to_low16(r[0]) | (even_bits_to_low16(r[1]) << 16);
        p0.y = even_bits_to_low16(r[2]) | (even_bits_to_low16(r[3]) << 16);
        p1.x = even_bits_to_low16(r[0] >> 1) | (even_bits_to_low16(r[1] >> 1) << 16);
        p1.y = even_bits_to_low16(r[2] >> 1) | (even_bits_to_low16(r[3] >> 1) << 16);
        uint32_t *row0 = planes + (((size_t)b * nchans_pad + c) * 2) * (size_t)row_pitch;
        *reinterpret_cast<uint2 *>(row0 + 2 * i) = p0;
        *reinterpret_cast<uint2 *>(row0 + row_pitch + 2 * i) = p1;
    }
}

// 8-bit samples: thread i of a row turns input bytes [32i, 32i+32) (32 samples) into
// one word of each of the 8 bit planes.  Three aligned 16-byte vectors cover the bytes.
__global__ void __launch_bounds__(128)
planes8_kernel(const uint8_t *__restrict__ in, size_t in_beam_stride, size_t row_stride,
               int nchans, const uint8_t *valid_begin, const uint8_t *valid_end,
               uint32_t *__restrict__ planes, int row_pitch, int nchans_pad)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;   // 32-sample word
    const int c = blockIdx.y, b = blockIdx.z;
    if (i >= row_pitch || c >= nchans_pad) return;
    uint32_t pw[8] = {0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u};
    const long long nvalid = (long long)row_stride - 32ll * i;
    if (c < nchans && nvalid > 0) {
        const uint8_t *a = in + (size_t)b * in_beam_stride + (size_t)c * row_stride + 32u * (size_t)i;
        const uintptr_t a0 = (uintptr_t)a & ~(uintptr_t)15;
        const int m = (int)((uintptr_t)a & 15);
        uint32_t v[12];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            uint4 q = make_uint4(0, 0, 0, 0);
            if (k < 2 || m) q = load_block16(a0 + 16u * k, valid_begin, valid_end);
            v[4 * k] = q.x; v[4 * k + 1] = q.y; v[4 * k + 2] = q.z; v[4 * k + 3] = q.w;
        }
        const int q4 = m >> 2, sh = (m & 3) * 8;
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            uint32_t x0 = v[k], x1 = v[k + 1];
            if (q4 == 1) { x0 = v[k + 1]; x1 = v[k + 2]; }
            if (q4 == 2) { x0 = v[k + 2]; x1 = v[k + 3]; }
            if (q4 == 3) { x0 = v[k + 3]; x1 = v[k + 4]; }
            uint32_t r = __funnelshift_r(x0, x1, sh);     // samples 4k .. 4k+3, one per byte
            const long long nb = nvalid - 4 * k;
            if (nb <= 0) r = 0;
            else if (nb < 4) r &= (1u << (8 * (int)nb)) - 1u;
            // bit p of the 4 bytes -> a nibble: the multiply gathers bits 0,8,16,24 into 24..27
#pragma unroll
            for (int p = 0; p < 8; ++p) {
                const uint32_t nib = (((r >> p) & 0x01010101u) * 0x01020408u) >> 24;
                pw[p] |= nib << (4 * k);
            }
        }
    }
    uint32_t *row0 = planes + (((size_t)b * nchans_pad + c) * 8) * (size_t)row_pitch;
#pragma unroll
    for (int p = 0; p < 8; ++p) row0[(size_t)p * row_pitch + i] = pw[p];
}

// ---- 1-bit and 4-bit samples (row f4) ----
// Bytes [16 i, 16 i + 16) of a tight row as four byte-aligned words (zero past the row end):
// the same two aligned 128-bit loads + funnel shifts as planes2_kernel.
__device__ __forceinline__ void load16_aligned(const uint8_t *a, long long nvalid,
                                               const uint8_t *valid_begin, const uint8_t *valid_end,
                                               uint32_t (&r)[4])
{
    const uintptr_t a0 = (uintptr_t)a & ~(uintptr_t)15;
    const int m = (int)((uintptr_t)a & 15);
    const uint4 lo = load_block16(a0, valid_begin, valid_end);
    const uint4 hi = m ? load_block16(a0 + 16, valid_begin, valid_end) : make_uint4(0, 0, 0, 0);
    const uint32_t v[8] = {lo.x, lo.y, lo.z, lo.w, hi.x, hi.y, hi.z, hi.w};
    const int q = m >> 2, sh = (m & 3) * 8;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        uint32_t x0 = v[k], x1 = v[k + 1];
        if (q == 1) { x0 = v[k + 1]; x1 = v[k + 2]; }
        if (q == 2) { x0 = v[k + 2]; x1 = v[k + 3]; }
        if (q == 3) { x0 = v[k + 3]; x1 = v[k + 4 < 8 ? k + 4 : 7]; }
        r[k] = __funnelshift_r(x0, x1, sh);
        const long long nb = nvalid - 4 * k;
        if (nb <= 0) r[k] = 0;
        else if (nb < 4) r[k] &= (1u << (8 * (int)nb)) - 1u;
    }
}

// bits 0, 4, 8, ..., 28 of x -> bits 0..7
__device__ __forceinline__ uint32_t every_fourth_bit_to_low8(uint32_t x)
{
    x &= 0x11111111u;
    x = (x | (x >> 3)) & 0x03030303u;
    x = (x | (x >> 6)) & 0x000f000fu;
    x = (x | (x >> 12)) & 0x000000ffu;
    return x;
}

// 1-bit: the LSB-first packed row IS bit plane 0; thread i copies 16 bytes = 4 words (128 samples).
__global__ void __launch_bounds__(128)
planes1_kernel(const uint8_t *__restrict__ in, size_t in_beam_stride, size_t row_stride,
               int nchans, const uint8_t *valid_begin, const uint8_t *valid_end,
               uint32_t *__restrict__ planes, int row_pitch, int nchans_pad)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;   // 128-sample block
    const int c = blockIdx.y, b = blockIdx.z;
    if (4 * i >= row_pitch || c >= nchans_pad) return;
    uint32_t r[4] = {0u, 0u, 0u, 0u};
    const long long nvalid = (long long)row_stride - 16ll * i;
    if (c < nchans && nvalid > 0)
        load16_aligned(in + (size_t)b * in_beam_stride + (size_t)c * row_stride + 16u * (size_t)i, nvalid,
                       valid_begin, valid_end, r);
    uint32_t *row0 = planes + ((size_t)b * nchans_pad + c) * (size_t)row_pitch;
    *reinterpret_cast<uint4 *>(row0 + 4 * i) = make_uint4(r[0], r[1], r[2], r[3]);
}

// 4-bit: thread i turns 16 bytes = 32 samples into one word of each of the 4 planes.
__global__ void __launch_bounds__(128)
planes4_kernel(const uint8_t *__restrict__ in, size_t in_beam_stride, size_t row_stride,
               int nchans, const uint8_t *valid_begin, const uint8_t *valid_end,
               uint32_t *__restrict__ planes, int row_pitch, int nchans_pad)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;   // 32-sample word
    const int c = blockIdx.y, b = blockIdx.z;
    if (i >= row_pitch || c >= nchans_pad) return;
    uint32_t r[4] = {0u, 0u, 0u, 0u};
    const long long nvalid = (long long)row_stride - 16ll * i;
    if (c < nchans && nvalid > 0)
        load16_aligned(in + (size_t)b * in_beam_stride + (size_t)c * row_stride + 16u * (size_t)i, nvalid,
                       valid_begin, valid_end, r);
    uint32_t *row0 = planes + (((size_t)b * nchans_pad + c) * 4) * (size_t)row_pitch;
#pragma unroll
    for (int p = 0; p < 4; ++p)
        row0[(size_t)p * row_pitch + i] =
            every_fourth_bit_to_low8(r[0] >> p) | (every_fourth_bit_to_low8(r[1] >> p) << 8) |
            (every_fourth_bit_to_low8(r[2] >> p) << 16) | (every_fourth_bit_to_low8(r[3] >> p) << 24);
}

cudaError_t launch_planes(int nbits, const uint8_t *in, size_t in_beam_stride, size_t row_stride,
                          int nchans, int nbeams, uint32_t *planes, int row_pitch, int nchans_pad,
                          cudaStream_t s)
{
    const uint8_t *vend = in + (size_t)(nbeams - 1) * in_beam_stride + (size_t)nchans * row_stride;
    if (nbits == 2) {
        dim3 block(128), grid((row_pitch / 2 + 127) / 128, nchans_pad, nbeams);
        planes2_kernel<<<grid, block, 0, s>>>(in, in_beam_stride, row_stride, nchans, in, vend, planes,
                                              row_pitch, nchans_pad);
    } else if (nbits == 1) {
        dim3 block(128), grid((row_pitch / 4 + 127) / 128, nchans_pad, nbeams);
        planes1_kernel<<<grid, block, 0, s>>>(in, in_beam_stride, row_stride, nchans, in, vend, planes,
                                              row_pitch, nchans_pad);
    } else if (nbits == 4) {
        dim3 block(128), grid((row_pitch + 127) / 128, nchans_pad, nbeams);
        planes4_kernel<<<grid, block, 0, s>>>(in, in_beam_stride, row_stride, nchans, in, vend, planes,
                                              row_pitch, nchans_pad);
    } else {
        dim3 block(128), grid((row_pitch + 127) / 128, nchans_pad, nbeams);
        planes8_kernel<<<grid, block, 0, s>>>(in, in_beam_stride, row_stride, nchans, in, vend, planes,
                                              row_pitch, nchans_pad);
    }
    ++g_launch_count;
    return cudaGetLastError();
}

// ---- time-scrunch pre-passes (row f4, reading R38) ----
// n low bits set in every `period` bits
__host__ __device__ constexpr uint32_t rep_mask(int n, int period)
{
    uint32_t m = 0;
    for (int b = 0; b < 32; ++b)
        if (b % period < n) m |= 1u << b;
    return m;
}

// bit i*F of x -> bit i  (32/F bits): log2(32/F) mask-shift steps
template <int F>
__device__ __forceinline__ uint32_t gather_every(uint32_t x)
{
    x &= rep_mask(1, F);
#pragma unroll
    for (int g = 1; g * F < 32; g *= 2) x = (x | (x >> (g * (F - 1)))) & rep_mask(2 * g, 2 * g * F);
    return x;
}

// Thread i of a row sums blocks of K = 2^LOG2K samples of NBITS bits and emits word i (32 block sums)
// of each of NPL bit planes.  F = NBITS*K <= 32 bits of the row make one sum, so the thread reads the
// F words from byte 4*F*i of the (tight, arbitrarily aligned) row: F+1 aligned 32-bit loads and a
// funnel shift.  Adjacent fields are added pairwise in place (SWAR, LOG2K steps; a sum of K samples
// fits its F-bit field), then bit p of every field is gathered into plane p.
template <int NBITS, int LOG2K, int NPL>
__global__ void __launch_bounds__(128)
planes_tscrunch_kernel(const uint8_t *__restrict__ in, size_t in_beam_stride, size_t row_stride,
                       int nchans, const uint8_t *valid_begin, const uint8_t *valid_end,
                       uint32_t *__restrict__ planes, int row_pitch, int nchans_pad)
{
    constexpr int F = NBITS << LOG2K;     // bits per block
    constexpr int PER = 32 / F;           // block sums per 32-bit word
    static_assert(F <= 32, "a block must fit one word");
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int c = blockIdx.y, b = blockIdx.z;
    if (i >= row_pitch || c >= nchans_pad) return;
    uint32_t pw[NPL];
#pragma unroll
    for (int p = 0; p < NPL; ++p) pw[p] = 0u;
    const long long nvalid = (long long)row_stride - 4ll * F * i;   // bytes of the row from this thread's first
    if (c < nchans && nvalid > 0) {
        const uint8_t *a = in + (size_t)b * in_beam_stride + (size_t)c * row_stride + (size_t)(4 * F) * (size_t)i;
        const uintptr_t a0 = (uintptr_t)a & ~(uintptr_t)3;
        const int sh = (int)((uintptr_t)a & 3) * 8;
        uint32_t v[F + 1];
#pragma unroll
        for (int q = 0; q <= F; ++q) {
            const uintptr_t aq = a0 + 4u * q;
            // an aligned word is loaded only if it overlaps the caller's buffer and the thread's bytes
            const bool need = (q < F || sh) && 4ll * q - (sh >> 3) < nvalid &&
                              aq + 4 > (uintptr_t)valid_begin && aq < (uintptr_t)valid_end;
            uint32_t word = 0u;
            if (need && aq >= (uintptr_t)valid_begin && aq + 4 <= (uintptr_t)valid_end) {
                word = __ldg(reinterpret_cast<const uint32_t *>(aq));
            } else if (need) {      // partial first / last word of the caller's buffer: byte loads inside it only
                for (int k = 0; k < 4; ++k)
                    if (aq + k >= (uintptr_t)valid_begin && aq + k < (uintptr_t)valid_end)
                        word |= (uint32_t)__ldg(reinterpret_cast<const uint8_t *>(aq + k)) << (8 * k);
            }
            v[q] = word;
        }
#pragma unroll
        for (int q = 0; q < F; ++q) {
            uint32_t x = __funnelshift_r(v[q], v[q + 1], sh);
            const long long nb = nvalid - 4 * q;
            if (nb <= 0) x = 0;
            else if (nb < 4) x &= (1u << (8 * (int)nb)) - 1u;
#pragma unroll
            for (int f = NBITS; f < F; f *= 2) x = (x & rep_mask(f, 2 * f)) + ((x >> f) & rep_mask(f, 2 * f));
#pragma unroll
            for (int p = 0; p < NPL; ++p)
                if (p < F) pw[p] |= gather_every<F>(x >> p) << ((q * PER) & 31);
        }
    }
    uint32_t *row0 = planes + (((size_t)b * nchans_pad + c) * NPL) * (size_t)row_pitch;
#pragma unroll
    for (int p = 0; p < NPL; ++p) row0[(size_t)p * row_pitch + i] = pw[p];
}

// Any factor k (k * (2^nbits - 1) <= 255): one byte per block sum, for the DIRECT kernel.
__global__ void __launch_bounds__(256)
tscrunch_bytes_kernel(const uint8_t *__restrict__ in, size_t in_beam_stride, size_t row_stride, int nbits, int k,
                      long long nsamps_scr, uint8_t *__restrict__ out)
{
    const long long u = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (u >= nsamps_scr) return;
    const int c = blockIdx.y, b = blockIdx.z;
    const uint8_t *row = in + (size_t)b * in_beam_stride + (size_t)c * row_stride;
    uint32_t acc = 0;
    for (int j = 0; j < k; ++j) {
        const long long bit = (u * k + j) * nbits;
        acc += (row[bit >> 3] >> (bit & 7)) & ((1u << nbits) - 1u);
    }
    out[((size_t)b * gridDim.y + c) * (size_t)nsamps_scr + (size_t)u] = (uint8_t)acc;
}

cudaError_t launch_planes_tscrunch(int nbits, int k, int nplanes, const uint8_t *in, size_t in_beam_stride,
                                   size_t row_stride, int nchans, int nbeams, uint32_t *planes,
                                   int row_pitch, int nchans_pad, cudaStream_t s)
{
    const uint8_t *vend = in + (size_t)(nbeams - 1) * in_beam_stride + (size_t)nchans * row_stride;
    const dim3 block(128), grid((row_pitch + 127) / 128, nchans_pad, nbeams);
    const int key = nbits * 100 + k;
#define TSC(NB, LK, NPL)                                                                                    \
    case NB * 100 + (1 << LK):                                                                              \
        if (nplanes != NPL) return cudaErrorInvalidValue;                                                   \
        planes_tscrunch_kernel<NB, LK, NPL><<<grid, block, 0, s>>>(in, in_beam_stride, row_stride, nchans,  \
                                                                   in, vend, planes, row_pitch, nchans_pad); \
        break;
    switch (key) {
        TSC(1, 1, 2) TSC(1, 2, 3) TSC(1, 3, 4) TSC(1, 4, 5)
        TSC(2, 1, 3) TSC(2, 2, 4) TSC(2, 3, 5) TSC(2, 4, 6)
        TSC(4, 1, 5) TSC(4, 2, 6) TSC(4, 3, 8)
        default: return cudaErrorInvalidValue;
    }
#undef TSC
    ++g_launch_count;
    return cudaGetLastError();
}

cudaError_t launch_tscrunch_bytes(int nbits, int k, const uint8_t *in, size_t in_beam_stride, size_t row_stride,
                                  int nchans, int nbeams, long long nsamps_scr, uint8_t *out, cudaStream_t s)
{
    const dim3 block(256), grid((unsigned)((nsamps_scr + 255) / 256), nchans, nbeams);
    tscrunch_bytes_kernel<<<grid, block, 0, s>>>(in, in_beam_stride, row_stride, nbits, k, nsamps_scr, out);
    ++g_launch_count;
    return cudaGetLastError();
}

// ---- host side of set_dm_list ------------------------------------------------
static void free_tables(BitsliceTables &T)
{
    cudaFree(T.d_rel);
    cudaFree(T.d_ws);
    cudaFree(T.d_order);
    T = BitsliceTables();
}

void bitslice_release(dedisp_plan p)
{
    if (p->tab[1].d_rel != p->tab[0].d_rel) free_tables(p->tab[1]);
    else p->tab[1] = BitsliceTables();
    free_tables(p->tab[0]);
    for (int i = 0; i < bs::NGEOM; ++i) p->geom[i] = BitsliceGeom();
}

template <class C>
static void fill_geom(BitsliceGeom &G, int nchans_pad, const BitsliceTables &T, int tab)
{
    G = BitsliceGeom();
    G.nbits = C::NB;
    G.nchans_pad = nchans_pad;
    G.ndm_pad = T.ngroups * 32;
    G.ngroups = T.ngroups;
    G.nplanes_acc = C::NP;
    G.tab = tab;
    // a thread reads words off + warp*W + j, j = 0..W  =>  off_max + TILE_WORDS + 1 words
    const int need = T.max_off + C::TILE_WORDS + 1;
    if (need <= C::WIN_S) G.win_words = C::WIN_S;
    else if (need <= C::WIN_L) G.win_words = C::WIN_L;
    else return;   // cannot happen once dms_per_group is 1 (max_off = 3); the DIRECT kernel would serve the plan
    G.usable = T.d_rel != nullptr;
}

// Build the tables with `dpg` trials per group; cudaSuccess and T filled, or an error and T empty.
static cudaError_t build_tables(dedisp_plan p, const std::vector<int32_t> &sorted_dms, int dpg, int nchans_pad,
                                BitsliceTables &T)
{
    const int ndm = p->ndm;
    const int ngroups = (ndm + dpg - 1) / dpg;
    std::vector<int32_t> lanes((size_t)ngroups * 32, -1);
    for (int i = 0; i < ndm; ++i) lanes[(size_t)(i / dpg) * 32 + i % dpg] = sorted_dms[i];
    T = BitsliceTables();
    T.ngroups = ngroups;
    T.dms_per_group = dpg;
    int *d_max = nullptr;
    const size_t nrows = (size_t)ngroups * nchans_pad;
    cudaError_t e = cudaMalloc(&T.d_order, sizeof(int32_t) * lanes.size());
    if (e == cudaSuccess) e = cudaMalloc(&T.d_ws, sizeof(int32_t) * nrows);
    if (e == cudaSuccess) e = cudaMalloc(&T.d_rel, sizeof(uint32_t) * nrows * 32);
    if (e == cudaSuccess) e = cudaMalloc(&d_max, sizeof(int));
    if (e == cudaSuccess) e = cudaMemset(d_max, 0, sizeof(int));
    if (e == cudaSuccess)
        e = cudaMemcpy(T.d_order, lanes.data(), sizeof(int32_t) * lanes.size(), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
        bitslice_tables_kernel<<<ngroups, 256>>>(p->d_delay, p->nchans, ndm, T.d_order, nchans_pad, T.d_ws,
                                                 T.d_rel, d_max);
        ++g_launch_count;
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpy(&T.max_off, d_max, sizeof(int), cudaMemcpyDeviceToHost);
    cudaFree(d_max);
    if (e != cudaSuccess) free_tables(T);
    return e;
}

dedisp_status bitslice_prepare(dedisp_plan p)
{
    const int ndm = p->ndm;
    const int nchans_pad = (p->nchans + bs::CH_PAD - 1) / bs::CH_PAD * bs::CH_PAD;
    // trial DMs sorted ascending (stable) -> lanes of a group have nearby, monotone delays
    std::vector<int32_t> sorted(ndm);
    std::iota(sorted.begin(), sorted.end(), 0);
    std::stable_sort(sorted.begin(), sorted.end(), [&](int a, int b) { return p->dms[a] < p->dms[b]; });
    p->order_identity = true;
    for (int i = 0; i < ndm; ++i) p->order_identity = p->order_identity && sorted[i] == i;
    // largest window offset each family of geometries can take: WIN_L - tile words - 1
    const int lim0 = std::min({bs::Cfg1::WIN_L - bs::Cfg1::TILE_WORDS, bs::Cfg2::WIN_L - bs::Cfg2::TILE_WORDS,
                               bs::Cfg3::WIN_L - bs::Cfg3::TILE_WORDS, bs::Cfg4::WIN_L - bs::Cfg4::TILE_WORDS,
                               bs::Cfg5::WIN_L - bs::Cfg5::TILE_WORDS}) - 1;
    const int lim1 = std::min(bs::Cfg6::WIN_L - bs::Cfg6::TILE_WORDS, bs::Cfg8::WIN_L - bs::Cfg8::TILE_WORDS) - 1;
    cudaError_t e = cudaSuccess;
    int dpg = 32;
    for (; dpg >= 1; dpg >>= 1) {       // 32 trials per group unless the DM steps are too coarse for the window
        e = build_tables(p, sorted, dpg, nchans_pad, p->tab[0]);
        if (e != cudaSuccess || p->tab[0].max_off <= lim0 || dpg == 1) break;
        free_tables(p->tab[0]);
    }
    if (e == cudaSuccess) {
        if (p->tab[0].max_off <= lim1) {
            p->tab[1] = p->tab[0];      // shared (bitslice_release frees it once)
        } else {
            for (dpg >>= 1; dpg >= 1; dpg >>= 1) {
                e = build_tables(p, sorted, dpg, nchans_pad, p->tab[1]);
                if (e != cudaSuccess || p->tab[1].max_off <= lim1 || dpg == 1) break;
                free_tables(p->tab[1]);
            }
        }
    }
    if (e != cudaSuccess) {
        p->last_cuda_error = (int)e;
        bitslice_release(p);
        return e == cudaErrorMemoryAllocation ? DEDISP_ERR_ALLOC : DEDISP_ERR_CUDA;
    }
    fill_geom<bs::Cfg1>(p->geom[1], nchans_pad, p->tab[0], 0);
    fill_geom<bs::Cfg2>(p->geom[2], nchans_pad, p->tab[0], 0);
    fill_geom<bs::Cfg3>(p->geom[3], nchans_pad, p->tab[0], 0);
    fill_geom<bs::Cfg4>(p->geom[4], nchans_pad, p->tab[0], 0);
    fill_geom<bs::Cfg5>(p->geom[5], nchans_pad, p->tab[0], 0);
    fill_geom<bs::Cfg6>(p->geom[6], nchans_pad, p->tab[1], 1);
    fill_geom<bs::Cfg8>(p->geom[8], nchans_pad, p->tab[1], 1);
    return DEDISP_OK;
}
