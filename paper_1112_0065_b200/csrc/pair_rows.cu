// pair_rows.cu -- set-up and pre-pass of the pair-row path of the tiled gather-sum (2-, 4- and 8-bit samples).
//
//   out[d][t] = sum_c in[c][t + delay[c][d]]                      (BASELINE.json:north_star)
//             = sum_p S_{p, delta_p(d)}[t + delay[2p][d]],   S_{p,delta}[u] = in[2p][u] + in[2p+1][u + delta],
//               delta_p(d) = delay[2p+1][d] - delay[2p][d]   (exact: the same integer sum, re-associated)
//
// Neighbouring trial DMs share delta_p, so the sum of a channel pair is formed ONCE per delay difference (a
// "pair row" of 3 bit planes, built by pair_rows_kernel from the 2-bit planes) instead of once per trial; the
// tiled kernel then adds nchans/2 three-plane rows per output sample instead of nchans two-plane rows.
//   * pair_range_kernel : the range of delta_p over the whole DM list -> the list of rows to build;
//   * pair_tables_kernel: per (DM group, pair) the first row the group's trials use, how many consecutive rows
//     (<= Cfg3P::NV, else the plan stays on the plain path), window start and per-lane offset/shift words;
//   * pair_rows_kernel  : the rows themselves, once per execute (a thread writes all rows of its pair for its
//     four words).
#include <vector>

#include "bitslice_common.cuh"
#include "dedisp_internal.h"

using namespace bs;

namespace {

// one warp per pair: min / max of delay[2p+1][d] - delay[2p][d] over all trials (0 for padding channels)
__global__ void pair_range_kernel(const int32_t *__restrict__ delay, int nchans, int ndm, int npairs,
                                  int32_t *__restrict__ dlo, int32_t *__restrict__ dhi)
{
    const int p = blockIdx.x, lane = threadIdx.x;
    if (p >= npairs) return;
    int lo = 0x7fffffff, hi = 0;
    if (2 * p + 1 < nchans) {
        const int32_t *d0 = delay + (size_t)(2 * p) * ndm, *d1 = d0 + ndm;
        for (int d = lane; d < ndm; d += 32) {
            const int v = d1[d] - d0[d];
            lo = min(lo, v);
            hi = max(hi, v);
        }
    } else {
        lo = 0;
    }
    for (int o = 16; o > 0; o >>= 1) {
        lo = min(lo, __shfl_xor_sync(0xffffffffu, lo, o));
        hi = max(hi, __shfl_xor_sync(0xffffffffu, hi, o));
    }
    if (lane == 0) {
        dlo[p] = lo;
        dhi[p] = hi;
    }
}

// One block per DM group, threads over pairs.  flags[0] = largest window offset (words), flags[1] = 1 when a
// (group, pair) needs more than nv consecutive rows.
__global__ void pair_tables_kernel(const int32_t *__restrict__ delay, int nchans, int ndm,
                                   const int32_t *__restrict__ sorted, int npairs_pad,
                                   const int32_t *__restrict__ dlo, const int32_t *__restrict__ row0, int nv,
                                   int slot_bytes, int skew_unit_bytes, int skew_odd_bytes, int32_t *__restrict__ ws, uint32_t *__restrict__ rel,
                                   uint32_t *__restrict__ vinfo, int *flags)
{
    const int g = blockIdx.x;
    int worst = 0;
    for (int p = threadIdx.x; p < npairs_pad; p += blockDim.x) {
        const size_t row = (size_t)g * npairs_pad + p;
        if (2 * p >= nchans) {
            ws[row] = 0;
            vinfo[row] = (uint32_t)row0[p];
            for (int l = 0; l < 32; ++l) rel[row * 32 + l] = 0;
            continue;
        }
        const int32_t *d0 = delay + (size_t)(2 * p) * ndm;
        const bool two = 2 * p + 1 < nchans;
        const int first = sorted[g * 32];
        const int w0 = (d0[first] >> 5) & ~3;
        ws[row] = w0;
        int lo = 0x7fffffff, hi = 0, last = first;
        for (int l = 0; l < 32; ++l) {
            const int d = sorted[g * 32 + l];
            if (d >= 0) last = d;
            const int v = two ? d0[ndm + last] - d0[last] : 0;
            lo = min(lo, v);
            hi = max(hi, v);
        }
        if (hi - lo + 1 > nv) {
            atomicOr(flags + 1, 1);
            hi = lo + nv - 1;
        }
        vinfo[row] = (uint32_t)(row0[p] + lo - dlo[p]) | ((uint32_t)(hi - lo) << 28);
        last = first;
        for (int l = 0; l < 32; ++l) {
            const int d = sorted[g * 32 + l];
            if (d >= 0) last = d;
            const int dv = d0[last];
            int v = (two ? d0[ndm + last] - dv : 0) - lo;
            v = v > nv - 1 ? nv - 1 : v;
            const int off = (dv >> 5) - w0;
            worst = max(worst, off);
            rel[row * 32 + l] = ((uint32_t)(off * 4 + v * slot_bytes + v * skew_unit_bytes + (v & 1) * skew_odd_bytes) << 16) | (uint32_t)(dv & 31);
        }
    }
    for (int o = 16; o > 0; o >>= 1) worst = max(worst, __shfl_xor_sync(0xffffffffu, worst, o));
    if ((threadIdx.x & 31) == 0) atomicMax(flags, worst);
}

// All rows of pair p (differences lo .. lo + n - 1, consecutive rows from row0): word w of the NB + 1 planes of
// row (p, delta) = planes of in[2p][u] + in[2p+1][u + delta] for the 32 samples u of word w (a bit-sliced ripple
// adder: NB full adders per word).  Thread = 4 consecutive words: the even channel is loaded once (128-bit
// loads), the odd channel's 5 words per plane at word offset delta >> 5 are re-read only when that offset
// changes and funnel-shifted by delta & 31 for every row, so a row costs its 128-bit stores and nothing else.
// (sweep on B200, pre-pass ms of the HTRU gulp / the 8-bit wideband: block 32 0.097 / 2.00, 64 0.094 / 1.83,
//  128 0.093 / 1.74, 128 with streaming stores 0.092 / 1.73, 64 with streaming stores 0.094 / 1.83)
#ifndef PAIR_ROWS_STCS
#define PAIR_ROWS_STCS 0
#endif
#if PAIR_ROWS_STCS
#define PAIR_ROWS_STORE(p, v) __stcs((p), (v))
#else
#define PAIR_ROWS_STORE(p, v) (*(p) = (v))
#endif
#ifndef PAIR_ROWS_BLOCK
#define PAIR_ROWS_BLOCK 128
#endif
template <int NB>
__global__ void __launch_bounds__(PAIR_ROWS_BLOCK)
pair_rows_kernel(const uint32_t *__restrict__ raw, size_t raw_beam_pitch, int nchans_pad,
                 const int32_t *__restrict__ pair_row0, const int32_t *__restrict__ pair_dlo,
                 const int32_t *__restrict__ pair_cnt, uint32_t *__restrict__ rows, size_t rows_beam_pitch,
                 int row_pitch)
{
    const int w = 4 * (blockIdx.y * blockDim.x + threadIdx.x);
    const int p = blockIdx.x, b = blockIdx.z;
    if (w >= row_pitch) return;
    const int lo = pair_dlo[p], n = pair_cnt[p];
    const size_t rstride = (size_t)(NB + 1) * row_pitch;
    uint32_t *dst = rows + (size_t)b * rows_beam_pitch + (size_t)pair_row0[p] * rstride + w;
    if (2 * p >= nchans_pad) {
        for (int i = 0; i < n; ++i, dst += rstride)
#pragma unroll
            for (int k = 0; k <= NB; ++k) *reinterpret_cast<uint4 *>(dst + (size_t)k * row_pitch) = make_uint4(0, 0, 0, 0);
        return;
    }
    const uint32_t *a = raw + (size_t)b * raw_beam_pitch + (size_t)(2 * p) * NB * row_pitch;
    const uint32_t *o = a + (size_t)NB * row_pitch;   // odd channel (nchans_pad is even)
    uint32_t x[NB][4], q[NB][5];
#pragma unroll
    for (int k = 0; k < NB; ++k) {
        const uint4 v = *reinterpret_cast<const uint4 *>(a + (size_t)k * row_pitch + w);
        x[k][0] = v.x; x[k][1] = v.y; x[k][2] = v.z; x[k][3] = v.w;
    }
    int cur = -1;
    for (int i = 0; i < n; ++i, dst += rstride) {
        const int delta = lo + i, sh = delta & 31;
        if ((delta >> 5) != cur) {
            cur = delta >> 5;
            const int wo = w + cur;
#pragma unroll
            for (int k = 0; k < NB; ++k)
#pragma unroll
                for (int j = 0; j < 5; ++j) q[k][j] = wo + j < row_pitch ? o[(size_t)k * row_pitch + wo + j] : 0u;
        }
        uint32_t c[4] = {0u, 0u, 0u, 0u};
#pragma unroll
        for (int k = 0; k < NB; ++k) {
            uint32_t s[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const uint32_t y = __funnelshift_r(q[k][j], q[k][j + 1], sh);
                s[j] = x[k][j] ^ y ^ c[j];
                c[j] = (x[k][j] & y) | (c[j] & (x[k][j] ^ y));
            }
            PAIR_ROWS_STORE(reinterpret_cast<uint4 *>(dst + (size_t)k * row_pitch), make_uint4(s[0], s[1], s[2], s[3]));
        }
        PAIR_ROWS_STORE(reinterpret_cast<uint4 *>(dst + (size_t)NB * row_pitch), make_uint4(c[0], c[1], c[2], c[3]));
    }
}

}  // namespace

static void release_tables(PairTables &T)
{
    cudaFree(T.d_rel);
    cudaFree(T.d_ws);
    cudaFree(T.d_vinfo);
    cudaFree(T.d_pair_row0);
    cudaFree(T.d_pair_dlo);
    cudaFree(T.d_pair_cnt);
    T = PairTables();
}

void pair_release(dedisp_plan p)
{
    release_tables(p->pairs);
    release_tables(p->pairs4);
    release_tables(p->pairs8);
}

// Called after bitslice_prepare: same DM groups as the raw geometry (B) and the windows of pair geometry C.  A
// plan the pair rows cannot serve (a group whose trials need more than C::NV differences of a pair, offsets
// beyond the window) leaves T.usable false; that is not an error.
template <class C>
static dedisp_status prepare_tables(dedisp_plan p, const BitsliceGeom &G2, const BitsliceTables &B, PairTables &T)
{
    release_tables(T);
    if (!G2.usable || !B.d_order || p->nchans < 2) return DEDISP_OK;
    const int npairs_pad = ((G2.nchans_pad / 2) + CH_PAD - 1) / CH_PAD * CH_PAD;
    const int ndm = p->ndm, ngroups = B.ngroups;
    int32_t *d_lo = nullptr, *d_hi = nullptr, *d_row0 = nullptr;
    int *d_flags = nullptr;
    std::vector<int32_t> lo(npairs_pad), hi(npairs_pad), row0(npairs_pad);
    cudaError_t e = cudaMalloc(&d_lo, sizeof(int32_t) * npairs_pad);
    if (e == cudaSuccess) e = cudaMalloc(&d_hi, sizeof(int32_t) * npairs_pad);
    if (e == cudaSuccess) e = cudaMalloc(&d_row0, sizeof(int32_t) * npairs_pad);
    if (e == cudaSuccess) e = cudaMalloc(&d_flags, 2 * sizeof(int));
    if (e == cudaSuccess) e = cudaMemset(d_flags, 0, 2 * sizeof(int));
    if (e == cudaSuccess) {
        pair_range_kernel<<<npairs_pad, 32>>>(p->d_delay, p->nchans, ndm, npairs_pad, d_lo, d_hi);
        ++g_launch_count;
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpy(lo.data(), d_lo, sizeof(int32_t) * npairs_pad, cudaMemcpyDeviceToHost);
    if (e == cudaSuccess) e = cudaMemcpy(hi.data(), d_hi, sizeof(int32_t) * npairs_pad, cudaMemcpyDeviceToHost);
    long long nrows = 0;
    bool fits = true;
    if (e == cudaSuccess) {
        for (int q = 0; q < npairs_pad; ++q) {
            row0[q] = (int32_t)nrows;
            nrows += (long long)hi[q] - lo[q] + 1;
            if (nrows > 0x07ffffff) { fits = false; break; }
        }
    }
    if (e == cudaSuccess && fits) {
        std::vector<int32_t> cnt(npairs_pad);
        for (int q = 0; q < npairs_pad; ++q) cnt[q] = hi[q] - lo[q] + 1;
        const size_t ntab = (size_t)ngroups * npairs_pad, pbytes = sizeof(int32_t) * npairs_pad;
        e = cudaMemcpy(d_row0, row0.data(), pbytes, cudaMemcpyHostToDevice);
        if (e == cudaSuccess) e = cudaMalloc(&T.d_pair_row0, pbytes);
        if (e == cudaSuccess) e = cudaMalloc(&T.d_pair_dlo, pbytes);
        if (e == cudaSuccess) e = cudaMalloc(&T.d_pair_cnt, pbytes);
        if (e == cudaSuccess) e = cudaMalloc(&T.d_ws, sizeof(int32_t) * ntab);
        if (e == cudaSuccess) e = cudaMalloc(&T.d_vinfo, sizeof(uint32_t) * ntab);
        if (e == cudaSuccess) e = cudaMalloc(&T.d_rel, sizeof(uint32_t) * ntab * 32);
        if (e == cudaSuccess) e = cudaMemcpy(T.d_pair_row0, row0.data(), pbytes, cudaMemcpyHostToDevice);
        if (e == cudaSuccess) e = cudaMemcpy(T.d_pair_dlo, lo.data(), pbytes, cudaMemcpyHostToDevice);
        if (e == cudaSuccess) e = cudaMemcpy(T.d_pair_cnt, cnt.data(), pbytes, cudaMemcpyHostToDevice);
        if (e == cudaSuccess) {
            pair_tables_kernel<<<ngroups, 256>>>(p->d_delay, p->nchans, ndm, B.d_order, npairs_pad, d_lo, d_row0,
                                                 C::NV, C::template vslot_words<C::WIN_S>() * 4, (C::vskew(2) - 2 * C::vskew(1) == 0 ? C::vskew(1) : 0) * 4,
                                                 (C::vskew(2) == 0 ? C::vskew(1) : 0) * 4, T.d_ws, T.d_rel, T.d_vinfo, d_flags);
            ++g_launch_count;
            e = cudaGetLastError();
        }
        int flags[2] = {0, 0};
        if (e == cudaSuccess) e = cudaMemcpy(flags, d_flags, sizeof(flags), cudaMemcpyDeviceToHost);
        if (e == cudaSuccess) {
            T.nrows = (int)nrows;
            T.npairs_pad = npairs_pad;
            T.usable = !flags[1] && flags[0] + C::TILE_WORDS + 1 <= C::WIN_S;
        }
    }
    cudaFree(d_lo);
    cudaFree(d_hi);
    cudaFree(d_row0);
    cudaFree(d_flags);
    if (e != cudaSuccess) {
        p->last_cuda_error = (int)e;
        release_tables(T);
        return e == cudaErrorMemoryAllocation ? DEDISP_ERR_ALLOC : DEDISP_ERR_CUDA;
    }
    if (!T.usable) release_tables(T);
    return DEDISP_OK;
}

dedisp_status pair_prepare(dedisp_plan p)
{
    dedisp_status st = prepare_tables<Cfg3P>(p, p->geom[2], p->tab[0], p->pairs);
    if (st == DEDISP_OK) st = prepare_tables<Cfg5P>(p, p->geom[4], p->tab[0], p->pairs4);
    if (st == DEDISP_OK) st = prepare_tables<Cfg9P>(p, p->geom[8], p->tab[1], p->pairs8);
    return st;
}

cudaError_t launch_pair_rows(const PairTables &T, int raw_nbits, const uint32_t *raw, size_t raw_beam_pitch,
                             int nchans_pad, uint32_t *rows, size_t rows_beam_pitch, int row_pitch, int nbeams,
                             cudaStream_t s)
{
    const dim3 block(PAIR_ROWS_BLOCK), grid(T.npairs_pad, (row_pitch / 4 + PAIR_ROWS_BLOCK - 1) / PAIR_ROWS_BLOCK, nbeams);
    if (raw_nbits == 2)
        pair_rows_kernel<2><<<grid, block, 0, s>>>(raw, raw_beam_pitch, nchans_pad, T.d_pair_row0, T.d_pair_dlo,
                                                   T.d_pair_cnt, rows, rows_beam_pitch, row_pitch);
    else if (raw_nbits == 4)
        pair_rows_kernel<4><<<grid, block, 0, s>>>(raw, raw_beam_pitch, nchans_pad, T.d_pair_row0, T.d_pair_dlo,
                                                   T.d_pair_cnt, rows, rows_beam_pitch, row_pitch);
    else
        pair_rows_kernel<8><<<grid, block, 0, s>>>(raw, raw_beam_pitch, nchans_pad, T.d_pair_row0, T.d_pair_dlo,
                                                   T.d_pair_cnt, rows, rows_beam_pitch, row_pitch);
    ++g_launch_count;
    return cudaGetLastError();
}
