// time_major.cu -- telescope-order (time-major, channel fastest) filterbank stream ->
// channel-major tight rows, the layout dedisp_execute reads (
// PAPER.md:20; reading R37).
//
//   in : sample (t, c) = bits [ (t*nchans + c)*nbits, +nbits ) of the stream, LSB-first
//   out: sample (c, t) = bits [ t*nbits, +nbits ) of row c, rows of ceil(nsamps*nbits/8) bytes
//
// A bit-level transpose, HBM-bound and small (the packed input of a gulp is 22 MB).  With
// E = 32/nbits samples per 32-bit word, a thread loads the same word column of E consecutive time
// samples (a warp reads 128 contiguous bytes of one time sample per load), transposes the E x E
// matrix of nbits-wide elements in registers (log2 E butterfly stages of masked XOR swaps) and
// thereby holds E output words: E consecutive time samples of each of its E channels.  A CTA
// gathers TS such steps per channel row in shared memory ([k][lane][step], odd pitch: conflict-free
// both ways) and writes every row segment (TS words = up to 128 contiguous bytes) with aligned
// 32-bit stores; rows are tight, so a row may start at any byte: the words are re-aligned with a
// funnel shift and only the first/last partial word of a segment is written byte by byte.
#include "dedisp_internal.h"

namespace {

// steps of E time samples per CTA (TS words = 4*TS bytes per channel row segment): 32 (1-bit: 16)
// for large streams, 8 when the grid would otherwise be a few waves only (measured on B200:
// gulp 2-bit 22 MB: TS 4/8/16/32 = 43.6/40.3/41.2/50.0 us; wide8 740 MB: 778/625/601/579 us)
__host__ __device__ constexpr int tm_steps_large(int nbits) { return nbits == 1 ? 16 : 32; }
constexpr int TM_STEPS_SMALL = 8;

template <int NBITS>
__device__ __forceinline__ void transpose_elems(uint32_t (&x)[32 / NBITS])
{
    constexpr int E = 32 / NBITS;
#pragma unroll
    for (int b = E / 2; b >= 1; b >>= 1) {
        const int shift = b * NBITS;
        // columns whose bit b is clear: blocks of `shift` bits, starting at bit 0
        const uint32_t mask = shift == 16 ? 0x0000ffffu : shift == 8 ? 0x00ff00ffu : shift == 4 ? 0x0f0f0f0fu
                            : shift == 2 ? 0x33333333u : 0x55555555u;
#pragma unroll
        for (int i = 0; i < E; ++i) {
            if (i & b) continue;
            const uint32_t t = ((x[i] >> shift) ^ x[i + b]) & mask;   // upper block of row i <-> lower block of row i+b
            x[i + b] ^= t;
            x[i] ^= t << shift;
        }
    }
}

// bytes [first, first+count) of the aligned word at p
__device__ __forceinline__ void store_some_bytes(uint8_t *p, uint32_t v, int first, int count)
{
    for (int q = first; q < first + count; ++q) p[q] = (uint8_t)(v >> (8 * q));
}

template <int NBITS, int TS>
__global__ void __launch_bounds__(256)
time_major_kernel(const uint32_t *__restrict__ in, int row_words, int nchans, long long nsamps,
                  uint8_t *__restrict__ out, size_t out_row_stride)
{
    constexpr int E = 32 / NBITS;
    constexpr int TSP = TS + 1;
    extern __shared__ uint32_t sm[];                      // [E][32][TSP]
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const long long t0 = (long long)blockIdx.x * (TS * E);
    const int wc0 = blockIdx.y * 32, wc = wc0 + lane;
    for (int step = warp; step < TS; step += 8) {
        uint32_t x[E];
        const long long tb = t0 + (long long)step * E;
        const long long left_t = nsamps - tb;
        const int nv = wc < row_words ? (left_t < E ? (int)left_t : E) : 0;      // valid time samples of the step
        const uint32_t *p = in + tb * row_words + wc;
#pragma unroll
        for (int i = 0; i < E; ++i) x[i] = i < nv ? __ldg(p + (size_t)i * row_words) : 0u;
        transpose_elems<NBITS>(x);
#pragma unroll
        for (int k = 0; k < E; ++k) sm[(k * 32 + lane) * TSP + step] = x[k];
    }
    __syncthreads();
    // ---- store phase ----
    const long long tile_byte0 = (long long)blockIdx.x * (TS * 4);
    const long long left = (long long)out_row_stride - tile_byte0;       // row bytes from this tile on
    const int nb = (int)(left < TS * 4 ? left : TS * 4);                 // valid bytes of the segment
    if (nb <= 0) return;
    // aligned global word j of row r holds segment bytes [4j - m, 4j - m + 4), m = row start & 3.
    // A warp writes 32 / TS rows per iteration, lane = (row, word j < TS): consecutive lanes read
    // consecutive shared words and store one contiguous run of TS aligned words per row.
    constexpr int RPI = 32 / TS;
    const int sub = lane / TS, j = lane % TS;
    const uint32_t *rowj = sm + (warp * RPI + sub) * TSP + j;            // word j of row (k = 0, lc0)
    const int cstep = 8 * RPI * E;                                       // channels between a warp's iterations
    if ((((uintptr_t)out | (uintptr_t)out_row_stride) & 3) == 0) {
        // every row starts on a word (rows of a multiple of 4 bytes): shared word j IS aligned global word j
        const bool full = 4 * j + 4 <= nb;
        const int tail = nb - 4 * j;                                     // 1..3: the row ends inside this word
        for (int k = 0; k < E; ++k) {
            int c = (wc0 + warp * RPI + sub) * E + k;
            uint8_t *dst = out + (size_t)c * out_row_stride + (size_t)tile_byte0 + 4 * j;
            const uint32_t *row = rowj + k * 32 * TSP;
#pragma unroll 4
            for (int it = 0; it < 32 / (8 * RPI); ++it, c += cstep, dst += (size_t)cstep * out_row_stride,
                     row += 8 * RPI * TSP) {
                if (c >= nchans) break;
                if (full) *reinterpret_cast<uint32_t *>(dst) = row[0];
                else if (tail > 0) store_some_bytes(dst, row[0], 0, tail);
            }
        }
        return;
    }
    for (int k = 0; k < E; ++k) {
        int c = (wc0 + warp * RPI + sub) * E + k;
        uint8_t *dst = out + (size_t)c * out_row_stride + (size_t)tile_byte0;
        const uint32_t *row = rowj + k * 32 * TSP;
#pragma unroll 4
        for (int it = 0; it < 32 / (8 * RPI); ++it, c += cstep, dst += (size_t)cstep * out_row_stride,
                 row += 8 * RPI * TSP) {
            if (c >= nchans) break;
            const int m = (int)((uintptr_t)dst & 3);
            const uint32_t hi = row[0], lo = j > 0 ? row[-1] : 0u;
            const uint32_t v = m ? __funnelshift_r(lo, hi, 8 * (4 - m)) : hi;
            const int s0 = 4 * j - m;                                    // segment byte of the word's byte 0
            const int first = s0 < 0 ? -s0 : 0;
            const int last = nb - s0 < 4 ? nb - s0 : 4;                  // exclusive, within the word
            if (last <= first) continue;
            if (first == 0 && last == 4) *reinterpret_cast<uint32_t *>(dst + s0) = v;
            else store_some_bytes(dst + s0, v, first, last - first);
        }
    }
    // the word after the last full one (segment bytes [4 TS - m, 4 TS)) exists only when m != 0
    for (int r = threadIdx.x; r < 32 * E; r += 256) {
        const long long c = (long long)(wc0 + (r & 31)) * E + (r >> 5);
        if (c >= nchans) continue;
        uint8_t *dst = out + (size_t)c * out_row_stride + (size_t)tile_byte0;
        const int m = (int)((uintptr_t)dst & 3);
        const int s0 = 4 * TS - m;
        const int last = nb - s0 < m ? nb - s0 : m;
        if (m == 0 || last <= 0) continue;
        store_some_bytes(dst + s0, sm[r * TSP + TS - 1] >> (8 * (4 - m)), 0, last);
    }
}

}  // namespace

extern "C" dedisp_status dedisp_transpose_time_major(const void *in_dev, int nchans, long long nsamps,
                                                     int nbits, void *out_dev, void *cuda_stream)
{
    if (!in_dev || !out_dev || nchans < 1 || nsamps < 1) return DEDISP_ERR_INVALID_ARG;
    if (nbits != 1 && nbits != 2 && nbits != 4 && nbits != 8) return DEDISP_ERR_UNSUPPORTED_NBITS;
    if (((long long)nchans * nbits) % 32 != 0 || ((uintptr_t)in_dev & 3u)) return DEDISP_ERR_INVALID_ARG;
    const int E = 32 / nbits;
    const int row_words = (int)((long long)nchans * nbits / 32);
    const int gy = (row_words + 31) / 32;
    int dev = 0, sms = 148;
    if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int TSL = tm_steps_large(nbits);
    const bool small = ((nsamps + (long long)TSL * E - 1) / ((long long)TSL * E)) * gy < 16ll * sms;
    const int TS = small ? TM_STEPS_SMALL : TSL;
    const long long gx = (nsamps + (long long)TS * E - 1) / ((long long)TS * E);
    if (gx > 0x7fffffffll || gy > 65535) return DEDISP_ERR_INVALID_ARG;
    const size_t stride = (size_t)(((unsigned long long)nsamps * (unsigned)nbits + 7) / 8);
    const size_t smem = (size_t)E * 32 * (TS + 1) * 4;
    const dim3 grid((unsigned)gx, (unsigned)gy), block(256);
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const uint32_t *in = (const uint32_t *)in_dev;
    uint8_t *out = (uint8_t *)out_dev;
    cudaError_t e = cudaSuccess;
#define TM_LAUNCH1(NB, T)                                                                               \
    do {                                                                                                \
        e = cudaFuncSetAttribute(time_major_kernel<NB, T>, cudaFuncAttributeMaxDynamicSharedMemorySize, \
                                 (int)smem);                                                            \
        if (e == cudaSuccess)                                                                           \
            time_major_kernel<NB, T><<<grid, block, smem, s>>>(in, row_words, nchans, nsamps, out, stride); \
    } while (0)
#define TM_LAUNCH(NB)                                      \
    do {                                                   \
        if (small) TM_LAUNCH1(NB, TM_STEPS_SMALL);         \
        else TM_LAUNCH1(NB, tm_steps_large(NB));           \
    } while (0)
    switch (nbits) {
        case 1: TM_LAUNCH(1); break;
        case 2: TM_LAUNCH(2); break;
        case 4: TM_LAUNCH(4); break;
        default: TM_LAUNCH(8); break;
    }
#undef TM_LAUNCH
#undef TM_LAUNCH1
    if (e != cudaSuccess) return DEDISP_ERR_CUDA;
    ++g_launch_count;
    return cudaGetLastError() == cudaSuccess ? DEDISP_OK : DEDISP_ERR_CUDA;
}
