// quad_rows.cu -- set-up and pre-pass of the quad-row path of the tiled gather-sum (8-bit samples).
//
//   out[d][t] = sum_c in[c][t + delay[c][d]]                      (BASELINE.json:north_star)
//             = sum_q Q_{q, D_q(d)}[t + delay[4q][d]],
//     Q_{q,(d1,d2,d3)}[u] = in[4q][u] + in[4q+1][u + d1] + in[4q+2][u + d2] + in[4q+3][u + d3],
//     D_q(d) = (delay[4q+k][d] - delay[4q][d])_{k = 1..3}          (exact: the same integer sum, re-associated)
//
// The step after the pair rows (pair_rows.cu): the sum of FOUR adjacent channels is formed once per triple of delay
// differences that occurs in the DM list (a "quad row" of nbits + 2 bit planes) and the tiled kernel adds nchans/4
// ten-plane rows per output sample instead of nchans/2 nine-plane rows: 0.59 x the adder and shift instructions of the
// pair-row kernel.  The price is memory and pre-pass traffic -- the 8-bit wideband config (4096 channels x 2048 trials)
// has 88 042 distinct (quad, triple) rows of 230 KB, 20.3 GB -- which is why only 8-bit data, where the gather-sum is
// slowest, takes this path (profiles/r2_wide8.md).
//   * quad_prepare      : (host bookkeeping on the DEVICE-built delay table) the distinct triples of every quad ->
//     the list of rows; per (DM group, quad) the <= NV rows the group's trials use, window start and per-lane
//     offset / shift / variant words.  More than NV distinct triples in a group, or offsets beyond the window: the
//     plan stays on the pair rows (not an error).
//   * quad_rows_kernel  : the rows themselves, once per execute, from the bit planes of the unpack pre-pass.
#include <algorithm>
#include <climits>
#include <cstdint>
#include <vector>

#include "bitslice_common.cuh"
#include "dedisp_internal.h"

using namespace bs;

namespace {

// All rows of quad q (triples in ascending (d1, d2, d3) order, consecutive rows from row0[q]): word w of the NB + 2
// planes of row (q; d1, d2, d3) for the 32 samples u of word w.  Thread = 4 consecutive words.  The partial sum
// in[4q] + in[4q+1][. + d1] (NB + 1 planes) is kept while d1 stays the same (it is the major sort key), channels 4q+2
// and 4q+3 are re-read (L1 / L2) and funnel-shifted for every row; additions are bit-sliced ripple adders.
#ifndef QUAD_ROWS_BLOCK
#define QUAD_ROWS_BLOCK 256
#endif
// y[k][0..4) = words [w, w + 4) of plane k of channel row `ch`, shifted down by delta samples (words beyond the row
// read as zero).  The five source words of a plane come from two ALIGNED 128-bit loads: the lanes of a warp read
// consecutive 16-byte pieces (one fully coalesced 512-byte request per load instead of five strided 32-bit ones --
// the 32-bit version ran at 95 % of the L1 throughput, profiles/r2_wide8.md), and which five of the eight words are
// used depends only on delta (the same for the whole block: no divergence).
template <int NB, int KK>
__device__ __forceinline__ void load_shifted_at(const uint32_t *__restrict__ ch, int row_pitch, int a, int sh,
                                                uint32_t (&y)[NB][4])
{
#pragma unroll
    for (int k = 0; k < NB; ++k) {
        const uint32_t *src = ch + (size_t)k * row_pitch + a;
        const uint4 lo = a < row_pitch ? __ldg(reinterpret_cast<const uint4 *>(src)) : make_uint4(0, 0, 0, 0);
        const uint4 hi = a + 4 < row_pitch ? __ldg(reinterpret_cast<const uint4 *>(src + 4)) : make_uint4(0, 0, 0, 0);
        const uint32_t q[8] = {lo.x, lo.y, lo.z, lo.w, hi.x, hi.y, hi.z, hi.w};
#pragma unroll
        for (int j = 0; j < 4; ++j) y[k][j] = __funnelshift_r(q[KK + j], q[KK + j + 1], sh);
    }
}

template <int NB>
__device__ __forceinline__ void load_shifted(const uint32_t *__restrict__ ch, int row_pitch, int w, int delta,
                                             uint32_t (&y)[NB][4])
{
    const int wo = w + (delta >> 5), sh = delta & 31, a = wo & ~3;     // row_pitch and w are multiples of 4
    switch (wo & 3) {
    case 0: load_shifted_at<NB, 0>(ch, row_pitch, a, sh, y); break;
    case 1: load_shifted_at<NB, 1>(ch, row_pitch, a, sh, y); break;
    case 2: load_shifted_at<NB, 2>(ch, row_pitch, a, sh, y); break;
    default: load_shifted_at<NB, 3>(ch, row_pitch, a, sh, y); break;
    }
}

// acc (NA planes) += y (NB planes), NB <= NA - 1: ripple through the planes of y, then the carry alone
template <int NA, int NB>
__device__ __forceinline__ void add_planes(uint32_t (&acc)[NA][4], const uint32_t (&y)[NB][4], int planes_in_use)
{
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        uint32_t c = 0;
#pragma unroll
        for (int k = 0; k < NA; ++k) {
            if (k < NB) {
                const uint32_t a = acc[k][j], b = y[k][j];
                acc[k][j] = a ^ b ^ c;
                c = (a & b) | (c & (a ^ b));
            } else if (k < planes_in_use) {
                const uint32_t a = acc[k][j];
                acc[k][j] = a ^ c;
                c = a & c;
            }
        }
    }
}

template <int NB>
__global__ void __launch_bounds__(QUAD_ROWS_BLOCK, 512 / QUAD_ROWS_BLOCK)
quad_rows_kernel(const uint32_t *__restrict__ raw, size_t raw_beam_pitch, int nchans_pad,
                 const int32_t *__restrict__ row0, const int4 *__restrict__ trip, uint32_t *__restrict__ rows,
                 size_t rows_beam_pitch, int row_pitch)
{
    constexpr int NR = NB + 2;
    const int w = 4 * (blockIdx.y * blockDim.x + threadIdx.x);
    const int q = blockIdx.x, b = blockIdx.z;
    if (w >= row_pitch) return;
    const int r0 = row0[q], r1 = row0[q + 1];
    const size_t rstride = (size_t)NR * row_pitch;
    uint32_t *dst = rows + (size_t)b * rows_beam_pitch + (size_t)r0 * rstride + w;
    if (4 * q + 3 >= nchans_pad) {       // (nchans_pad is a multiple of 32: cannot happen; rows of padding quads are zero)
        for (int r = r0; r < r1; ++r, dst += rstride)
#pragma unroll
            for (int k = 0; k < NR; ++k) *reinterpret_cast<uint4 *>(dst + (size_t)k * row_pitch) = make_uint4(0, 0, 0, 0);
        return;
    }
    const uint32_t *c0 = raw + (size_t)b * raw_beam_pitch + (size_t)(4 * q) * NB * row_pitch;
    const uint32_t *c1 = c0 + (size_t)NB * row_pitch, *c2 = c1 + (size_t)NB * row_pitch, *c3 = c2 + (size_t)NB * row_pitch;
    uint32_t s01[NR][4];       // in[4q] + in[4q+1][. + d1]: NB + 1 planes in use
    int cur_d1 = -1;
    for (int r = r0; r < r1; ++r, dst += rstride) {
        const int4 t = __ldg(trip + r);
        if (t.x != cur_d1) {
            cur_d1 = t.x;
#pragma unroll
            for (int k = 0; k < NR; ++k) {
                uint4 v = make_uint4(0, 0, 0, 0);
                if (k < NB) v = __ldg(reinterpret_cast<const uint4 *>(c0 + (size_t)k * row_pitch + w));
                s01[k][0] = v.x; s01[k][1] = v.y; s01[k][2] = v.z; s01[k][3] = v.w;
            }
            uint32_t y[NB][4];
            load_shifted<NB>(c1, row_pitch, w, t.x, y);
            add_planes<NR, NB>(s01, y, NB + 1);
        }
        uint32_t acc[NR][4];
#pragma unroll
        for (int k = 0; k < NR; ++k)
#pragma unroll
            for (int j = 0; j < 4; ++j) acc[k][j] = s01[k][j];
        {
            uint32_t y[NB][4];
            load_shifted<NB>(c2, row_pitch, w, t.y, y);
            add_planes<NR, NB>(acc, y, NR);
        }
        {
            uint32_t y[NB][4];
            load_shifted<NB>(c3, row_pitch, w, t.z, y);
            add_planes<NR, NB>(acc, y, NR);
        }
#pragma unroll
        for (int k = 0; k < NR; ++k) {
            const uint4 o = make_uint4(acc[k][0], acc[k][1], acc[k][2], acc[k][3]);
            // streaming store: 20.3 GB of rows pass through L2 once; evict-first keeps the channel planes, which every
            // row of the quad re-reads, resident (pre-pass 5.57 -> 4.75 ms on the 8-bit wideband config)
            __stcs(reinterpret_cast<uint4 *>(dst + (size_t)k * row_pitch), o);
        }
    }
}

void release_tables(QuadTables &T)
{
    cudaFree(T.d_rel);
    cudaFree(T.d_ws);
    cudaFree(T.d_vlist);
    cudaFree(T.d_row0);
    cudaFree(T.d_trip);
    T = QuadTables();
}

}  // namespace

void quad_release(dedisp_plan p) { release_tables(p->quads8); }

// The host half of quad_prepare, on HOST copies of the delay table [nchans][ndm] and of the lane order
// [ngroups][32] (output row of each lane, -1 = padding): pure bookkeeping, no CUDA call -- also reachable without a GPU
// through dedisp_debug_quad_tables (tests/test_quad_tables_cpu.py checks the addressing contract of the tables).
struct QuadHost {
    std::vector<int32_t> row0, ws, trip;
    std::vector<int2> vlist;
    std::vector<uint32_t> rel;
    long long nrows = 0;
    bool fits = false;
};

template <class C>
static void build_tables_host(const int32_t *delay, const int32_t *lanes, int nchans, int ndm, int ngroups,
                              int nquads_pad, QuadHost &H)
{
    constexpr int NV = C::NV;
    constexpr int VSLOT_BYTES = C::template vslot_words<C::WIN_S>() * 4;
    constexpr int PLW = C::template plane_words<C::WIN_S>();      // words of one plane line of a staged box
    constexpr int PMAX = PLW - C::TILE_WORDS - 1;                 // last box word a lane's window may start at
    static_assert(VSLOT_BYTES % 128 == 0, "the variant slots start at bank 0");
    std::vector<int32_t> &row0 = H.row0, &ws = H.ws, &trip = H.trip;
    std::vector<int2> &vlist = H.vlist;
    std::vector<uint32_t> &rel = H.rel;
    row0.assign(nquads_pad + 1, 0);
    ws.assign((size_t)ngroups * nquads_pad, 0);
    vlist.assign((size_t)ngroups * nquads_pad * NV, make_int2(-1, 0));
    rel.assign((size_t)ngroups * nquads_pad * 32, 0u);
    trip.clear();
    std::vector<uint64_t> keys(ndm), uniq;
    bool fits = true;
    long long nrows = 0;
    // A TMA box must start on a 16-byte boundary of global memory: box starts that are not a multiple of 4 words fault
    // with "illegal instruction" on sm_100a (measured, profiles/r2_wide8.md), so the placement moves in steps of 4.
    constexpr int gran = 4;
    for (int q = 0; q < nquads_pad && fits; ++q) {
        row0[q] = (int32_t)nrows;
        if (4 * q >= nchans) {       // padding quad: one all-zero row (triple 0, 0, 0), windows at 0
            trip.insert(trip.end(), {0, 0, 0, 0});
            for (int g = 0; g < ngroups; ++g) vlist[((size_t)g * nquads_pad + q) * NV] = make_int2((int32_t)nrows, 0);
            ++nrows;
            continue;
        }
        const int32_t *d0 = &delay[(size_t)(4 * q) * ndm];
        auto diff = [&](int k, int d) -> int64_t {      // channels beyond nchans are all-zero rows: difference 0
            return 4 * q + k < nchans ? (int64_t)delay[(size_t)(4 * q + k) * ndm + d] - d0[d] : 0;
        };
        for (int d = 0; d < ndm && fits; ++d) {
            const int64_t a = diff(1, d), b = diff(2, d), c = diff(3, d);
            if (a < 0 || b < 0 || c < 0 || a >= (1 << 20) || b >= (1 << 20) || c >= (1 << 20)) fits = false;
            keys[d] = ((uint64_t)a << 40) | ((uint64_t)b << 20) | (uint64_t)c;
        }
        if (!fits) break;
        uniq = keys;
        std::sort(uniq.begin(), uniq.end());
        uniq.erase(std::unique(uniq.begin(), uniq.end()), uniq.end());
        for (uint64_t k : uniq)
            trip.insert(trip.end(), {(int32_t)(k >> 40), (int32_t)((k >> 20) & 0xfffff), (int32_t)(k & 0xfffff), 0});
        for (int g = 0; g < ngroups && fits; ++g) {
            const size_t slot = (size_t)g * nquads_pad + q;
            // the variant (row) and the window word of every lane
            int used[NV], nused = 0, lv[32], lw[32], ld[32], last = lanes[(size_t)g * 32];
            for (int l = 0; l < 32 && fits; ++l) {
                const int d = lanes[(size_t)g * 32 + l];
                if (d >= 0) last = d;       // padding lanes repeat the group's last trial
                const int id = (int)(std::lower_bound(uniq.begin(), uniq.end(), keys[last]) - uniq.begin());
                int v = 0;
                while (v < nused && used[v] != id) ++v;
                if (v == nused) {
                    if (nused == NV) { fits = false; break; }
                    used[nused++] = id;
                }
                lv[l] = v;
                ld[l] = d0[last];
                lw[l] = d0[last] >> 5;
            }
            if (!fits) break;
            ws[slot] = *std::min_element(lw, lw + 32);
            // Every variant gets a box start of its own: box word (lw - wmin_v + s_v) holds the lane's first word.
            // The triples of neighbouring trials alternate, so the variants' windows interleave; s_v is chosen (greedy,
            // in order of first use) so that the distinct words the 32 lanes read in one shared-memory load fall into
            // as many different banks as possible (same word = broadcast; the variant slots start at bank 0; plane
            // and tile-word offsets are common to all lanes).  Average wavefronts per load on the 8-bit wideband list:
            // 1.64 with a fixed skew per variant, 1.30 with this placement (profiles/r2_wide8.md).
            int occ[32] = {};
            for (int v = 0; v < nused && fits; ++v) {
                int wmin = INT32_MAX, wmax = INT32_MIN;
                for (int l = 0; l < 32; ++l)
                    if (lv[l] == v) { wmin = std::min(wmin, lw[l]); wmax = std::max(wmax, lw[l]); }
                const int span = wmax - wmin;
                if (span > PMAX) { fits = false; break; }
                uint32_t seen[4] = {};      // distinct words of this variant, relative to wmin (span <= PMAX < 128)
                for (int l = 0; l < 32; ++l)
                    if (lv[l] == v) seen[(lw[l] - wmin) >> 5] |= 1u << ((lw[l] - wmin) & 31);
                int best_s = 0, best_max = INT32_MAX, best_hits = INT32_MAX;
                for (int sft = 0; sft <= PMAX - span && sft < 32 + gran; ++sft) {
                    if ((wmin - sft) & (gran - 1)) continue;
                    int mx = 0, hits = 0;
                    int add[32] = {};
                    for (int o = 0; o <= span; ++o)
                        if (seen[o >> 5] >> (o & 31) & 1u) ++add[(o + sft) & 31];
                    for (int bk = 0; bk < 32; ++bk) {
                        mx = std::max(mx, occ[bk] + add[bk]);
                        hits += occ[bk] * add[bk] + add[bk] * (add[bk] - 1) / 2;
                    }
                    if (mx < best_max || (mx == best_max && hits < best_hits)) { best_max = mx; best_hits = hits; best_s = sft; }
                    if (mx <= 1) break;      // no two words share a bank: cannot be improved
                }
                for (int o = 0; o <= span; ++o)
                    if (seen[o >> 5] >> (o & 31) & 1u) ++occ[(o + best_s) & 31];
                vlist[slot * NV + v] = make_int2((int32_t)(nrows + used[v]), wmin - best_s);
                for (int l = 0; l < 32; ++l)
                    if (lv[l] == v)
                        rel[slot * 32 + l] = ((uint32_t)((lw[l] - wmin + best_s) * 4 + v * VSLOT_BYTES) << 16) | (uint32_t)(ld[l] & 31);
            }
        }
        nrows += (long long)uniq.size();
        if (nrows > 0x03ffffff) fits = false;
    }
    row0[nquads_pad] = (int32_t)nrows;
    H.nrows = nrows;
    H.fits = fits;
}

// Called after pair_prepare.  Host bookkeeping on the delay table the device built (copied back once per set_dm_list):
// differences, de-duplication and indices only -- no arithmetic of the method.  Leaves T.usable false (not an error)
// when the plan cannot take quad rows.
template <class C>
static dedisp_status prepare_tables(dedisp_plan p, const BitsliceGeom &G, const BitsliceTables &B, QuadTables &T)
{
    release_tables(T);
    if (!G.usable || !B.d_order || p->nchans < 4 || B.dms_per_group < 1) return DEDISP_OK;
    const int ndm = p->ndm, nchans = p->nchans, ngroups = B.ngroups;
    const int nquads_pad = ((G.nchans_pad / 4) + CH_PAD - 1) / CH_PAD * CH_PAD;
    const size_t tbl = (size_t)nchans * ndm;
    if (tbl > ((size_t)1 << 28) || (size_t)ngroups * nquads_pad * 32 > ((size_t)1 << 28)) return DEDISP_OK;   // host budget
    std::vector<int32_t> delay(tbl), lanes((size_t)ngroups * 32);
    cudaError_t e = cudaMemcpy(delay.data(), p->d_delay, tbl * sizeof(int32_t), cudaMemcpyDeviceToHost);
    if (e == cudaSuccess) e = cudaMemcpy(lanes.data(), B.d_order, lanes.size() * sizeof(int32_t), cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) {
        p->last_cuda_error = (int)e;
        return DEDISP_ERR_CUDA;
    }
    QuadHost H;
    build_tables_host<C>(delay.data(), lanes.data(), nchans, ndm, ngroups, nquads_pad, H);
    constexpr int NV = C::NV;
    const bool fits = H.fits;
    const long long nrows = H.nrows;
    std::vector<int32_t> &row0 = H.row0, &ws = H.ws, &trip = H.trip;
    std::vector<int2> &vlist = H.vlist;
    std::vector<uint32_t> &rel = H.rel;
    if (!fits) return DEDISP_OK;
    const size_t ntab = (size_t)ngroups * nquads_pad;
    e = cudaMalloc(&T.d_rel, ntab * 32 * sizeof(uint32_t));
    if (e == cudaSuccess) e = cudaMalloc(&T.d_ws, ntab * sizeof(int32_t));
    if (e == cudaSuccess) e = cudaMalloc(&T.d_vlist, ntab * NV * sizeof(int2));
    if (e == cudaSuccess) e = cudaMalloc(&T.d_row0, (nquads_pad + 1) * sizeof(int32_t));
    if (e == cudaSuccess) e = cudaMalloc(&T.d_trip, trip.size() * sizeof(int32_t));
    if (e == cudaSuccess) e = cudaMemcpy(T.d_rel, rel.data(), ntab * 32 * sizeof(uint32_t), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(T.d_ws, ws.data(), ntab * sizeof(int32_t), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(T.d_vlist, vlist.data(), ntab * NV * sizeof(int2), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(T.d_row0, row0.data(), (nquads_pad + 1) * sizeof(int32_t), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(T.d_trip, trip.data(), trip.size() * sizeof(int32_t), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) {
        cudaGetLastError();
        p->last_cuda_error = (int)e;
        release_tables(T);
        return e == cudaErrorMemoryAllocation ? DEDISP_ERR_ALLOC : DEDISP_ERR_CUDA;
    }
    T.nrows = (int)nrows;
    T.nquads_pad = nquads_pad;
    T.usable = true;
    return DEDISP_OK;
}

// include/dedisp.h: the tables of the quad-row path from host arrays, no GPU involved
extern "C" dedisp_status dedisp_debug_quad_tables(int nchans, int ndm, const int *delay_host, int ngroups,
                                                  const int *lanes_host, dedisp_quad_table_info *info, int *row0,
                                                  int *trip, int *vlist, unsigned int *rel)
{
    using C = Cfg10Q;
    if (!delay_host || !lanes_host || !info || nchans < 4 || ndm < 1 || ngroups < 1) return DEDISP_ERR_INVALID_ARG;
    const int nchans_pad = (nchans + CH_PAD - 1) / CH_PAD * CH_PAD;
    const int nquads_pad = ((nchans_pad / 4) + CH_PAD - 1) / CH_PAD * CH_PAD;
    if ((size_t)nchans * ndm > ((size_t)1 << 28) || (size_t)ngroups * nquads_pad * 32 > ((size_t)1 << 28))
        return DEDISP_ERR_INVALID_ARG;
    for (int g = 0; g < ngroups; ++g) {
        if (lanes_host[(size_t)g * 32] < 0) return DEDISP_ERR_INVALID_ARG;
        for (int l = 0; l < 32; ++l)
            if (lanes_host[(size_t)g * 32 + l] >= ndm) return DEDISP_ERR_INVALID_ARG;
    }
    QuadHost H;
    build_tables_host<C>(delay_host, lanes_host, nchans, ndm, ngroups, nquads_pad, H);
    info->nv = C::NV;
    info->vslot_bytes = C::template vslot_words<C::WIN_S>() * 4;
    info->plane_words = C::template plane_words<C::WIN_S>();
    info->tile_words = C::TILE_WORDS;
    info->nquads_pad = nquads_pad;
    info->nrows = H.fits ? (int)H.nrows : 0;
    info->usable = H.fits ? 1 : 0;
    if (!H.fits) return DEDISP_OK;
    if (row0) std::copy(H.row0.begin(), H.row0.end(), row0);
    if (trip) std::copy(H.trip.begin(), H.trip.end(), trip);
    if (vlist)
        for (size_t i = 0; i < H.vlist.size(); ++i) {
            vlist[2 * i] = H.vlist[i].x;
            vlist[2 * i + 1] = H.vlist[i].y;
        }
    if (rel) std::copy(H.rel.begin(), H.rel.end(), rel);
    return DEDISP_OK;
}

dedisp_status quad_prepare(dedisp_plan p)
{
    // only where the pair rows already serve the plan (same DM groups, 8-bit window family) and the list is long
    // enough for the rows to pay: a handful of groups cannot amortise ~75 rows per quad
    release_tables(p->quads8);
    if (!p->pairs8.usable || p->tab[1].ngroups < 8) return DEDISP_OK;
    // one channel block only: sums of more than (2^NP - 1) / 255 = 4112 channels need the channel-block form of the
    // launch (execute_quads has it, as execute_pairs does), which no GPU test of the quad path has exercised -- such
    // plans stay on the pair rows, whose channel blocks are tested
    constexpr long long QUADS_PER_BLOCK = (((1ll << Cfg10Q::NP) - 1) / (4 * 255)) / CH_PAD * CH_PAD;
    if (((p->geom[8].nchans_pad / 4) + CH_PAD - 1) / CH_PAD * CH_PAD > QUADS_PER_BLOCK) return DEDISP_OK;
    return prepare_tables<Cfg10Q>(p, p->geom[8], p->tab[1], p->quads8);
}

cudaError_t launch_quad_rows(const QuadTables &T, int raw_nbits, const uint32_t *raw, size_t raw_beam_pitch,
                             int nchans_pad, uint32_t *rows, size_t rows_beam_pitch, int row_pitch, int nbeams,
                             cudaStream_t s)
{
    if (raw_nbits != 8) return cudaErrorInvalidValue;
    const dim3 block(QUAD_ROWS_BLOCK), grid(T.nquads_pad, (row_pitch / 4 + QUAD_ROWS_BLOCK - 1) / QUAD_ROWS_BLOCK, nbeams);
    quad_rows_kernel<8><<<grid, block, 0, s>>>(raw, raw_beam_pitch, nchans_pad, T.d_row0,
                                               reinterpret_cast<const int4 *>(T.d_trip), rows, rows_beam_pitch, row_pitch);
    ++g_launch_count;
    return cudaGetLastError();
}
