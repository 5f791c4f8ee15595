// time_major.cu -- telescope-order (time-major, channel fastest) filterbank stream ->
// channel-major tight rows, the layout dedisp_execute reads (
// PAPER.md:20; reading R37).
//
//   in : sample (t, c) = bits [ (t*nchans + c)*nbits, +nbits ) of the stream, LSB-first
//   out: sample (c, t) = bits [ t*nbits, +nbits ) of row c, rows of ceil(nsamps*nbits/8) bytes
//
// A bit-level transpose through shared memory, HBM-bound and small (the packed input of a
// gulp is 22 MB): a CTA takes a tile of 32 stream bytes (256/nbits channels) x 256 (1-bit: 128) time
// samples, reads it with 32-bit loads (32-byte segments per time sample), unpacks to one byte
// per sample in shared memory ([t][c], conflict-free writes), and each thread then packs the
// bytes of one output row segment.
#include "dedisp_internal.h"

namespace {

__host__ __device__ constexpr int tile_times(int nbits) { return nbits == 1 ? 128 : 256; }   // time samples per tile (<= 48 KB)
constexpr int TILE_BYTES = 32;     // stream bytes per time sample per tile

template <int NBITS>
__global__ void __launch_bounds__(256)
time_major_kernel(const uint32_t *__restrict__ in, int nchans, long long nsamps, uint8_t *__restrict__ out,
                  size_t out_row_stride)
{
    constexpr int TT = tile_times(NBITS);
    constexpr int SPB = 8 / NBITS;                 // samples per byte
    constexpr int CC = TILE_BYTES * SPB;           // channels per tile
    constexpr int PITCH = CC + 4;                  // bytes; keeps 32-bit alignment, staggers banks
    __shared__ __align__(4) uint8_t tile[TT * PITCH];
    const long long t0 = (long long)blockIdx.x * TT;
    const int c0 = blockIdx.y * CC;
    const int row_words = nchans * NBITS / 32;     // stream words per time sample
    const int tile_words = min(TILE_BYTES / 4, row_words - blockIdx.y * (TILE_BYTES / 4));
    const int nt = (int)min((long long)TT, nsamps - t0);
    // ---- load + unpack: word q of time sample t holds channels c0 + q*32/NBITS ... ----
    for (int idx = threadIdx.x; idx < nt * (TILE_BYTES / 4); idx += 256) {
        const int t = idx / (TILE_BYTES / 4), q = idx % (TILE_BYTES / 4);
        if (q >= tile_words) continue;
        const uint32_t w = __ldg(in + (t0 + t) * row_words + blockIdx.y * (TILE_BYTES / 4) + q);
        uint8_t *dst = tile + t * PITCH + q * (32 / NBITS);
        if (NBITS == 8) {
            *reinterpret_cast<uint32_t *>(dst) = w;
        } else {
#pragma unroll
            for (int k = 0; k < 32 / NBITS; k += 4) {
                const uint32_t a = (w >> (k * NBITS)) & ((1u << NBITS) - 1u);
                const uint32_t b = (w >> ((k + 1) * NBITS)) & ((1u << NBITS) - 1u);
                const uint32_t c = (w >> ((k + 2) * NBITS)) & ((1u << NBITS) - 1u);
                const uint32_t d = (w >> ((k + 3) * NBITS)) & ((1u << NBITS) - 1u);
                *reinterpret_cast<uint32_t *>(dst + k) = a | (b << 8) | (c << 16) | (d << 24);
            }
        }
    }
    __syncthreads();
    // ---- pack along time: consecutive threads write consecutive bytes of one channel row ----
    const int out_bytes = (nt * NBITS + 7) / 8;            // bytes of this tile per channel row
    const int ncl = min(CC, nchans - c0);
    for (int idx = threadIdx.x; idx < ncl * out_bytes; idx += 256) {
        const int cl = idx / out_bytes, bt = idx % out_bytes;
        uint32_t v = 0;
#pragma unroll
        for (int k = 0; k < SPB; ++k) {
            const int t = bt * SPB + k;
            if (t < nt) v |= (uint32_t)tile[t * PITCH + cl] << (k * NBITS);
        }
        out[(size_t)(c0 + cl) * out_row_stride + (size_t)(t0 * NBITS / 8) + bt] = (uint8_t)v;
    }
}

}  // namespace

extern "C" dedisp_status dedisp_transpose_time_major(const void *in_dev, int nchans, long long nsamps,
                                                     int nbits, void *out_dev, void *cuda_stream)
{
    if (!in_dev || !out_dev || nchans < 1 || nsamps < 1) return DEDISP_ERR_INVALID_ARG;
    if (nbits != 1 && nbits != 2 && nbits != 4 && nbits != 8) return DEDISP_ERR_UNSUPPORTED_NBITS;
    if (((long long)nchans * nbits) % 32 != 0 || ((uintptr_t)in_dev & 3u)) return DEDISP_ERR_INVALID_ARG;
    const int TT = tile_times(nbits);
    const long long gx = (nsamps + TT - 1) / TT;
    const int cc = TILE_BYTES * 8 / nbits;
    const int gy = (nchans + cc - 1) / cc;
    if (gx > 0x7fffffffll || gy > 65535) return DEDISP_ERR_INVALID_ARG;
    const size_t stride = (size_t)(((unsigned long long)nsamps * (unsigned)nbits + 7) / 8);
    const dim3 grid((unsigned)gx, (unsigned)gy), block(256);
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const uint32_t *in = (const uint32_t *)in_dev;
    uint8_t *out = (uint8_t *)out_dev;
    switch (nbits) {
        case 1: time_major_kernel<1><<<grid, block, 0, s>>>(in, nchans, nsamps, out, stride); break;
        case 2: time_major_kernel<2><<<grid, block, 0, s>>>(in, nchans, nsamps, out, stride); break;
        case 4: time_major_kernel<4><<<grid, block, 0, s>>>(in, nchans, nsamps, out, stride); break;
        default: time_major_kernel<8><<<grid, block, 0, s>>>(in, nchans, nsamps, out, stride); break;
    }
    ++g_launch_count;
    return cudaGetLastError() == cudaSuccess ? DEDISP_OK : DEDISP_ERR_CUDA;
}
