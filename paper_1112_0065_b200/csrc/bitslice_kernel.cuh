// bitslice_kernel.cuh -- kernel C: the tiled gather-sum (north_star subsystem (c), (d)).
//
//   out[d][t] = sum_c in[c][t + delay[c][d]]       (BASELINE.json:north_star)
//
// B200 design (the numbers are those of the 2-bit geometry Cfg2, see bitslice_common.cuh):
//   * a work item = (beam, group of 32 trial DMs, tile of 1920 output samples);
//     persistent CTAs (one per SM) walk the item list;
//   * lane  = trial DM, warp = 4 consecutive 32-sample words, 15 consumer warps;
//   * one producer warp stages, per 32-channel chunk, the window of bit-plane words
//     the tile needs with 1-D TMA bulk copies (cp.async.bulk + mbarrier tx counts)
//     into a 3-deep shared-memory ring, so neighbouring DMs reuse one staged window;
//   * consumers never unpack to integers: a sample stays 2 bit planes, is aligned
//     with one funnel shift per plane-word and is added with carry-save adders
//     (2 LOP3 per full adder) into a 12-plane bit-sliced counter held in registers
//     -- 32 additions per instruction, ~0.2 ALU ops per (channel, DM, sample);
//   * the counter is un-sliced once per tile and written as uint32 / float32;
//   * pair rows (Cfg3P / Cfg5P / Cfg9P, pair_rows.cu): the same kernel on rows that hold the sum of two
//     adjacent channels at a fixed delay difference (one more plane, half as many rows per tile), the
//     1-3 rows a DM group uses of a pair staged as 2-D TMA boxes (cp.async.bulk.tensor.2d).
#pragma once
#include <cuda.h>

#include <atomic>
#include <cmath>

#include "bitslice_common.cuh"
#include "dedisp_internal.h"

using namespace bs;

// This header is the whole templated kernel and its launchers; it is instantiated by one translation unit per
// geometry (bitslice_inst_*.cu, compiled in parallel) and dispatched by bitslice_kernel.cu.

namespace bsk {

__device__ __forceinline__ uint32_t smem_u32(const void *p)
{
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint32_t bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra DONE;\n"
        "bra LAB_WAIT;\n"
        "DONE:\n"
        "}\n" ::"r"(bar),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
        "l"(src), "r"(bytes), "r"(bar)
        : "memory");
}

// one 2-D box (plane lines x words) of the pair rows, through the tensor map
__device__ __forceinline__ void tma_box_g2s(uint32_t dst, const CUtensorMap *tm, int x, int y, uint32_t bar)
{
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(dst),
        "l"(tm), "r"(x), "r"(y), "r"(bar)
        : "memory");
}

// full adder on 32 independent bit positions: acc <- acc ^ x ^ y, returns majority(acc, x, y)
__device__ __forceinline__ uint32_t full_add(uint32_t &acc, uint32_t x, uint32_t y)
{
    uint32_t carry, sum;
    asm("lop3.b32 %0, %1, %2, %3, 0xE8;" : "=r"(carry) : "r"(acc), "r"(x), "r"(y));
    asm("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(sum) : "r"(acc), "r"(x), "r"(y));
    acc = sum;
    return carry;
}

template <class C, int WIN>
struct Stage {
    static constexpr int PLW = C::template plane_words<WIN>();         // words per plane line in the slot
    static constexpr int VSLOT = C::template vslot_words<WIN>() * 4;   // bytes per variant: [plane][PLW]
    static constexpr int BOX_BYTES = C::NB * PLW * 4;                  // bytes one TMA box delivers (NV > 1)
    static constexpr int CPITCH = C::NV * VSLOT;                       // bytes per channel slot
    static constexpr int DATA_BYTES = C::CH * CPITCH;
    static constexpr int REL_BYTES = C::CH * LANES * 4;
    static constexpr int BYTES = DATA_BYTES + REL_BYTES;
    static constexpr int SMEM = C::NSTAGE * BYTES + 2 * C::NSTAGE * 8 + C::NSTAGE * 8;   // ring, barriers, check tags
};

#ifdef DEDISP_CHECKS
__device__ __forceinline__ void check_fail(unsigned long long *errs, int code)
{
    if (errs) {
        atomicAdd(errs + CHK_TOTAL, 1ull);
        atomicAdd(errs + code, 1ull);
    }
}
#define BS_CHECK(cond, code) do { if (!(cond)) check_fail(P.check_errors, (code)); } while (0)
#else
#define BS_CHECK(cond, code) do { } while (0)
#endif

// Load the W+1 words of every plane of channel CI that this thread's W output words
// need, and align them to the output time axis (one funnel shift per plane-word).
// Geometries with many plane subsets (NSPLIT > 2) visit every channel slot once per subset: they keep the slot's
// rel word and window address in registers for the whole chunk (SlotCache) instead of re-deriving them per subset.
template <class C>
struct SlotCache {
    static constexpr bool ON = C::NSPLIT > 2;
    uint32_t r[ON ? C::CH : 1];
    const uint32_t *wp[ON ? C::CH : 1];
};

template <class C, int CI, int WIN, int P0>
__device__ __forceinline__ void load_aligned(const uint8_t *tb, const uint32_t *relp, const SlotCache<C> &sc,
                                             uint32_t (&x)[C::NBS][C::W])
{
    uint32_t r;
    const uint32_t *wp;
    if constexpr (SlotCache<C>::ON) {
        r = sc.r[CI];
        wp = sc.wp[CI] + P0 * Stage<C, WIN>::PLW;
    } else {
        r = relp[CI * LANES];
        wp = reinterpret_cast<const uint32_t *>(tb + (r >> 16)) + CI * (Stage<C, WIN>::CPITCH / 4) + P0 * Stage<C, WIN>::PLW;
    }
#pragma unroll
    for (int p = 0; p < C::NBS; ++p) {
        uint32_t w[C::W + 1];
#pragma unroll
        for (int j = 0; j <= C::W; ++j) w[j] = wp[p * Stage<C, WIN>::PLW + j];
#pragma unroll
        for (int j = 0; j < C::W; ++j) x[p][j] = __funnelshift_r(w[j], w[j + 1], r);   // shift = r & 31
    }
}

// Tree<K> adds planes P0 .. P0+NBS-1 of 2^(K+1) channels (C0 ...) into counter planes P0 .. P0+K+NBS-1 and
// hands back NBS carry words e[i] of weight 2^(P0+K+1+i): carry-save all the way, no ripple.
template <class C, int K, int C0, int WIN, int P0>
struct Tree {
    static __device__ __forceinline__ void run(uint32_t (&A)[C::NP][C::W], const uint8_t *tb,
                                               const uint32_t *relp, const SlotCache<C> &sc, uint32_t (&e)[C::NBS][C::W])
    {
        uint32_t e1[C::NBS][C::W], e2[C::NBS][C::W];
        Tree<C, K - 1, C0, WIN, P0>::run(A, tb, relp, sc, e1);
        Tree<C, K - 1, C0 + (1 << K), WIN, P0>::run(A, tb, relp, sc, e2);
#pragma unroll
        for (int i = 0; i < C::NBS; ++i)
#pragma unroll
            for (int j = 0; j < C::W; ++j) e[i][j] = full_add(A[P0 + K + i][j], e1[i][j], e2[i][j]);
    }
};
template <class C, int C0, int WIN, int P0>
struct Tree<C, 0, C0, WIN, P0> {
    static __device__ __forceinline__ void run(uint32_t (&A)[C::NP][C::W], const uint8_t *tb,
                                               const uint32_t *relp, const SlotCache<C> &sc, uint32_t (&e)[C::NBS][C::W])
    {
        uint32_t x0[C::NBS][C::W], x1[C::NBS][C::W];
        load_aligned<C, C0, WIN, P0>(tb, relp, sc, x0);
        load_aligned<C, C0 + 1, WIN, P0>(tb, relp, sc, x1);
#pragma unroll
        for (int i = 0; i < C::NBS; ++i)   // bit P0 + i of both channels
#pragma unroll
            for (int j = 0; j < C::W; ++j) e[i][j] = full_add(A[P0 + i][j], x0[i][j], x1[i][j]);
    }
};

// One chunk of CH channels: the tree of plane subset S, its NBS carry words added into the planes above
// the tree.  The subsets occupy adjacent plane ranges (subset S + 1 starts where the carries of subset S end),
// so the carry out of one subset's addition is the carry IN of the next one's: one chain through the counter
// per chunk instead of one ripple to the top plane per subset (8-bit pair rows, three subsets: 33 instead of
// 81 instructions per chunk and word, profiles/r2_wide8.md); only the last subset ripples into the top planes.
template <class C, int WIN, int S>
__device__ __forceinline__ void add_chunk(uint32_t (&A)[C::NP][C::W], const uint8_t *tb, const uint32_t *relp,
                                          const SlotCache<C> &sc, uint32_t (&c)[C::W])
{
    constexpr int P0 = S * C::NBS, B = P0 + C::K + 1, NBS = C::NBS, NP = C::NP, W = C::W;
    uint32_t e[NBS][W];
    Tree<C, C::K, 0, WIN, P0>::run(A, tb, relp, sc, e);
#pragma unroll
    for (int j = 0; j < W; ++j) {
        uint32_t cj;
        if constexpr (S == 0) {
            cj = A[B][j] & e[0][j];
            A[B][j] ^= e[0][j];
        } else {
            cj = full_add(A[B][j], e[0][j], c[j]);   // c: weight 2^B, handed over by subset S - 1
        }
#pragma unroll
        for (int i = 1; i < NBS; ++i) cj = full_add(A[B + i][j], e[i][j], cj);
        if constexpr (S + 1 < C::NSPLIT) {
            c[j] = cj;                               // carry in of the next subset
        } else {                                     // last subset: ripple into the top planes (word by word: one
#pragma unroll                                       // live carry register, as before the subsets were chained)
            for (int p = B + NBS; p < NP - 1; ++p) {
                const uint32_t t = A[p][j] & cj;
                A[p][j] ^= cj;
                cj = t;
            }
            if (B + NBS < NP) A[NP - 1][j] ^= cj;
        }
    }
    if constexpr (S + 1 < C::NSPLIT) add_chunk<C, WIN, S + 1>(A, tb, relp, sc, c);
}

// Work-item order (P.gblock): blocks of gblock DM groups; inside a block consecutive items are the
// groups of one time tile, so CTAs running at the same time stage overlapping windows of the planes
// (L2 hits) when the planes do not fit L2.  gblock = 1: consecutive items = consecutive tiles of a group.
__device__ __forceinline__ void item_coords(const BitsliceParams &P, long long item, int &beam, int &g, int &tile)
{
    const long long per_beam = (long long)P.ngroups * P.ntiles;
    beam = (int)(item / per_beam);
    const long long r = item - (long long)beam * per_beam;
    const long long per_blk = (long long)P.gblock * P.ntiles;
    const int blk = (int)(r / per_blk);
    const int g0 = blk * P.gblock;
    const int gb = P.ngroups - g0 < P.gblock ? P.ngroups - g0 : P.gblock;
    const int rr = (int)(r - (long long)blk * per_blk);
    tile = rr / gb;
    g = P.g_begin + g0 + rr - tile * gb;
}

// Transpose step of the un-slice: rows a (index i, i & s == 0) and b (index i + s)
// exchange the bit blocks (i, j | s) <-> (i + s, j).  m selects columns with j & s == 0.
__device__ __forceinline__ void swap_block(uint32_t &a, uint32_t &b, int s, uint32_t m)
{
    const uint32_t bs = b << s, as = a >> s;
    const uint32_t na = (a & m) | (bs & ~m);
    b = (b & ~m) | (as & m);
    a = na;
}

template <bool F32>
__device__ __forceinline__ uint32_t cvt_out(uint32_t v)
{
    // exact for v < 2^23: 2^23 + v is representable, subtracting 2^23 leaves float(v)
    return F32 ? __float_as_uint(__uint_as_float(v | 0x4B000000u) - 8388608.0f) : v;
}

// Un-slice one word (32 samples) of the counter and store it.  NP <= 16: the planes
// are transposed as two 16x16 bit blocks side by side (M[i] = out[i] | out[i+16] << 16);
// NP > 16: a full 32x32 transpose.
template <int NP, int W, bool F32>
__device__ __forceinline__ void unslice_store(uint32_t (&A)[NP][W], int j, uint8_t *orow, long long t0,
                                              long long nsamps_out, bool fast, bool accumulate)
{
    constexpr int R = (NP <= 16) ? 16 : 32;
    uint32_t M[R];
#pragma unroll
    for (int i = 0; i < R; ++i) M[i] = (i < NP) ? A[i][j] : 0u;
    if (R == 32) {
#pragma unroll
        for (int i = 0; i < 16; ++i) swap_block(M[i], M[i + 16], 16, 0x0000FFFFu);
    }
#pragma unroll
    for (int i = 0; i < R; ++i)
        if ((i & 8) == 0) swap_block(M[i], M[i + 8], 8, 0x00FF00FFu);
#pragma unroll
    for (int i = 0; i < R; ++i)
        if ((i & 4) == 0) swap_block(M[i], M[i + 4], 4, 0x0F0F0F0Fu);
#pragma unroll
    for (int i = 0; i < R; ++i)
        if ((i & 2) == 0) swap_block(M[i], M[i + 2], 2, 0x33333333u);
#pragma unroll
    for (int i = 0; i < R; ++i)
        if ((i & 1) == 0) swap_block(M[i], M[i + 1], 1, 0x55555555u);
    uint32_t o[32];
#pragma unroll
    for (int i = 0; i < 32; ++i) {
        if (R == 32) o[i] = M[i];
        else o[i] = (i < 16) ? (M[i] & 0xFFFFu) : (M[i - 16] >> 16);
    }
    if (accumulate) {
        // a later channel block: add the uint32 partial sums the earlier blocks left in out; the total
        // may reach 2^24 - 1, beyond the magic-number conversion, so convert with I2F here
        if (fast) {
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                const uint4 old = *reinterpret_cast<const uint4 *>(orow + (size_t)(t0 + 4 * q) * 4);
                o[4 * q] += old.x; o[4 * q + 1] += old.y; o[4 * q + 2] += old.z; o[4 * q + 3] += old.w;
            }
        } else {
#pragma unroll
            for (int i = 0; i < 32; ++i)
                if (t0 + i < nsamps_out) o[i] += *reinterpret_cast<const uint32_t *>(orow + (size_t)(t0 + i) * 4);
        }
#pragma unroll
        for (int i = 0; i < 32; ++i)
            if (F32) o[i] = __float_as_uint((float)o[i]);
    } else {
#pragma unroll
        for (int i = 0; i < 32; ++i) o[i] = cvt_out<F32>(o[i]);
    }
    if (fast) {
#pragma unroll
        for (int q = 0; q < 8; ++q)
            *reinterpret_cast<uint4 *>(orow + (size_t)(t0 + 4 * q) * 4) =
                make_uint4(o[4 * q], o[4 * q + 1], o[4 * q + 2], o[4 * q + 3]);
    } else {
#pragma unroll
        for (int i = 0; i < 32; ++i)
            if (t0 + i < nsamps_out) *reinterpret_cast<uint32_t *>(orow + (size_t)(t0 + i) * 4) = o[i];
    }
}

template <class C, int WIN, bool F32>
__global__ void __launch_bounds__(C::NTHREADS, 1) bitslice_dedisperse(const BitsliceParams P, const __grid_constant__ CUtensorMap tmap)
{
    constexpr int NW = C::NW, W = C::W, NP = C::NP, NB = C::NB, CH = C::CH, NSTAGE = C::NSTAGE;
    extern __shared__ __align__(128) uint8_t smem[];
    using S = Stage<C, WIN>;
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem + NSTAGE * S::BYTES);
    const uint32_t full0 = smem_u32(bars), empty0 = smem_u32(bars + NSTAGE);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
#ifdef DEDISP_CHECKS
    volatile long long *tags = reinterpret_cast<volatile long long *>(bars + 2 * NSTAGE);   // (item, chunk) in each stage
#endif
    if (threadIdx.x == 0) {
        for (int s = 0; s < NSTAGE; ++s) {
            mbar_init(full0 + 8 * s, 1);
            mbar_init(empty0 + 8 * s, NW);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const int nchunks = P.nchunks;
    const long long nitems = (long long)P.nbeams * P.ngroups * P.ntiles;
    int stage = 0;
    uint32_t phase = 0;

    if (warp == NW) {
        // ---------------- producer warp: TMA bulk copies into the ring ----------------
        for (long long item = blockIdx.x; item < nitems; item += gridDim.x) {
            int beam, g, tile;
            item_coords(P, item, beam, g, tile);
            const uint32_t *pl = P.planes + (size_t)beam * P.beam_pitch_words + (size_t)tile * C::TILE_WORDS;
            const size_t grow = (size_t)g * P.nchans_pad;
            for (int chunk = 0; chunk < nchunks; ++chunk) {
                mbar_wait(empty0 + 8 * stage, phase ^ 1);
                const uint32_t sb = smem_u32(smem) + stage * S::BYTES;
                const uint32_t fb = full0 + 8 * stage;
#ifdef DEDISP_CHECKS
                if (lane == 0)      // ordered before the arrive on full[] below
                    tags[stage] = (P.inject_fault == 1 && item == blockIdx.x && chunk == 0) ? -1 : item * nchunks + chunk;
                __syncwarp();
#endif
                if constexpr (C::NV == 1) {
                    if (lane == 0) mbar_expect_tx(fb, S::BYTES);
                    __syncwarp();
                    // one copy per (channel, plane) of the chunk, spread over the lanes
#pragma unroll
                    for (int i = lane; i < CH * NB; i += 32) {
                        const int c = (P.chunk0 + chunk) * CH + i / NB, pidx = i % NB;
                        const uint32_t *src = pl + ((size_t)c * NB + pidx) * P.row_pitch + P.ws[grow + c];
                        BS_CHECK(src >= P.planes && src + WIN <= P.planes + P.scratch_words && ((uintptr_t)src & 15) == 0 &&
                                     P.ws[grow + c] + tile * C::TILE_WORDS + WIN <= P.row_pitch, CHK_TMA_SRC);
                        bulk_g2s(sb + i * (WIN * 4), src, WIN * 4, fb);
                    }
                } else {
                    // pair rows: one box (NB plane lines x PLW words) per (channel slot, variant the group uses)
                    static_assert(C::NV == 1 || CH <= 32, "one lane per channel slot counts the variants");
                    const size_t c0 = grow + (size_t)(P.chunk0 + chunk) * CH;
                    if constexpr (C::NV > 3) {
                        // quad rows: lane = (slot, variant); the row of each variant is listed explicitly
                        static_assert(C::NV <= 3 || CH * C::NV <= 32, "one lane per (slot, variant)");
                        const int cl = lane / C::NV, v = lane % C::NV;
                        const int2 vr = lane < CH * C::NV ? P.vlist[(c0 + cl) * C::NV + v] : make_int2(-1, 0);
                        const int row = vr.x;
                        const int nbox = __reduce_add_sync(0xffffffffu, row >= 0 ? 1 : 0);
                        if (lane == 0) mbar_expect_tx(fb, S::REL_BYTES + nbox * S::BOX_BYTES);
                        __syncwarp();
                        if (row >= 0) {
                            // (the box may start before the row or run past its end: those words are zero-filled and
                            // never read -- the lanes' own words lie inside, quad_rows.cu::prepare_tables)
                            const int x = vr.y + tile * C::TILE_WORDS;
                            const int y = (beam * P.vrows + row) * NB;
                            BS_CHECK(x > -S::PLW && x < P.row_pitch && y >= 0 && (x & 3) == 0 &&
                                         (unsigned long long)(y + NB) * P.row_pitch <= P.scratch_words, CHK_TMA_SRC);
                            tma_box_g2s(sb + cl * S::CPITCH + v * S::VSLOT, &tmap, x, y, fb);
                        }
                    } else {
                    const int mine = lane < CH ? (int)(P.vinfo[c0 + lane] >> 28) + 1 : 0;
                    const int nbox = __reduce_add_sync(0xffffffffu, mine);
                    if (lane == 0) mbar_expect_tx(fb, S::REL_BYTES + nbox * S::BOX_BYTES);
                    __syncwarp();
#pragma unroll
                    for (int i = lane; i < CH * C::NV; i += 32) {
                        const int cl = i / C::NV, v = i % C::NV;
                        const uint32_t info = P.vinfo[c0 + cl];
                        if (v <= (int)(info >> 28)) {
                            const int x = P.ws[c0 + cl] + tile * C::TILE_WORDS - C::vskew(v);
                            const int y = (beam * P.vrows + (int)(info & 0x0fffffffu) + v) * NB;
                            // (x < 0 only by the designed skew of the variants: those words are zero-filled and never read)
                            BS_CHECK(x >= -C::VSKEW && x + S::PLW <= P.row_pitch && y >= 0 &&
                                         (unsigned long long)(y + NB) * P.row_pitch <= P.scratch_words && (x & 3) == 0, CHK_TMA_SRC);
                            tma_box_g2s(sb + cl * S::CPITCH + v * S::VSLOT, &tmap, x, y, fb);
                        }
                    }
                    }
                }
                if (lane == 0)
                    bulk_g2s(sb + S::DATA_BYTES, P.rel + (grow + (size_t)(P.chunk0 + chunk) * CH) * LANES,
                             S::REL_BYTES, fb);
                if (++stage == NSTAGE) { stage = 0; phase ^= 1; }
            }
        }
        return;
    }

    // ---------------- consumer warps ----------------
    uint32_t A[NP][W];
#pragma unroll
    for (int p = 0; p < NP; ++p)
#pragma unroll
        for (int j = 0; j < W; ++j) A[p][j] = 0;

    for (long long item = blockIdx.x; item < nitems; item += gridDim.x) {
        for (int chunk = 0; chunk < nchunks; ++chunk) {
            mbar_wait(full0 + 8 * stage, phase);
            const uint8_t *sb = smem + stage * S::BYTES;
            const uint8_t *tb = sb + warp * (W * 4);
            const uint32_t *relp = reinterpret_cast<const uint32_t *>(sb + S::DATA_BYTES) + lane;
#ifdef DEDISP_CHECKS
            BS_CHECK(tags[stage] == item * nchunks + chunk, CHK_STAGE_TAG);
            for (int ci = 0; ci < CH; ++ci) {
                // words read by load_aligned: byte offset of the lane + the slot + the warp's words, W + 1 words of NB planes
                const uint32_t first = (relp[ci * LANES] >> 16) + ci * S::CPITCH + warp * (W * 4);
                const uint32_t last = first + ((NB - 1) * S::PLW + W) * 4 + 4;
                BS_CHECK((first & 3) == 0 && last <= (uint32_t)S::DATA_BYTES && last <= (uint32_t)(ci + 1) * S::CPITCH, CHK_LDS_RANGE);
            }
#endif
            uint32_t carry[W];
            SlotCache<C> sc;
            if constexpr (SlotCache<C>::ON) {
#pragma unroll
                for (int ci = 0; ci < CH; ++ci) {
                    sc.r[ci] = relp[ci * LANES];
                    sc.wp[ci] = reinterpret_cast<const uint32_t *>(tb + (sc.r[ci] >> 16)) + ci * (S::CPITCH / 4);
                }
            }
            add_chunk<C, WIN, 0>(A, tb, relp, sc, carry);
#ifdef DEDISP_CHECKS
            BS_CHECK(tags[stage] == item * nchunks + chunk, CHK_STAGE_TAG);   // not overwritten while it was being read
#endif
            __syncwarp();
            if (lane == 0) mbar_arrive(empty0 + 8 * stage);
            if (++stage == NSTAGE) { stage = 0; phase ^= 1; }
        }

        // ---------------- epilogue: un-slice the counter, convert, store ----------------
        int beam, g, tile;
        item_coords(P, item, beam, g, tile);
        const int d = P.order[g * LANES + lane];
        BS_CHECK(d >= -1 && d < P.ndm && beam >= 0 && beam < P.nbeams, CHK_OUT_RANGE);
        uint8_t *orow = P.out + (size_t)beam * P.out_beam_stride +
                        (size_t)(d < 0 ? 0 : d) * (size_t)P.nsamps_out * 4;
#pragma unroll
        for (int j = 0; j < W; ++j) {
            const long long t0 = (long long)tile * C::TILE_SAMPS + (warp * W + j) * 32;
            if (d >= 0 && t0 < P.nsamps_out)
                unslice_store<NP, W, F32>(A, j, orow, t0, P.nsamps_out,
                                          P.vec_ok && t0 + 32 <= P.nsamps_out, P.accumulate != 0);
#pragma unroll
            for (int p = 0; p < NP; ++p) A[p][j] = 0;
        }
    }
}

template <class C, int WIN, bool F32>
cudaError_t launch_one(const BitsliceParams &P, int grid, cudaStream_t s, int device, const CUtensorMap *tm = nullptr)
{
    static const CUtensorMap no_map = {};
    constexpr int SMEM = Stage<C, WIN>::SMEM;
    static std::atomic<unsigned long long> attr_done{0};   // the attribute is per device: one bit per device id
    const unsigned long long bit = 1ull << (device & 63);
    if (device > 63 || !(attr_done.load(std::memory_order_acquire) & bit)) {
        cudaError_t e = cudaFuncSetAttribute(bitslice_dedisperse<C, WIN, F32>,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM);
        if (e != cudaSuccess) return e;
        attr_done.fetch_or(bit, std::memory_order_release);   // (setting it twice from two threads is harmless)
    }
    bitslice_dedisperse<C, WIN, F32><<<grid, C::NTHREADS, SMEM, s>>>(P, tm ? *tm : no_map);
    ++g_launch_count;
    return cudaGetLastError();
}

template <class C>
dedisp_status execute_cfg(dedisp_plan plan, const BitsliceGeom &G, int nbeams, long long nsamps_out,
                          const uint8_t *in, size_t row_stride, size_t in_beam_stride, int in_nbits,
                          int tscrunch, void *out, size_t out_beam_stride, int out_f32, cudaStream_t s,
                          const BitsliceRange &range, bool reserve_only)
{
    const long long ntiles = (nsamps_out + C::TILE_SAMPS - 1) / C::TILE_SAMPS;
    const long long pitch =
        (((long long)(plan->max_delay >> 5) + ntiles * C::TILE_WORDS + G.win_words + 4) + 3) & ~3ll;
    if (ntiles > 0x7fffffff / C::TILE_WORDS || pitch > 0x7fffffff) return DEDISP_ERR_INVALID_ARG;
    const size_t beam_pitch = (size_t)G.nchans_pad * C::NB * (size_t)pitch;
    const size_t need = beam_pitch * (size_t)nbeams * 4;
    if (G.nchans_pad > 65535 || nbeams > 65535) return DEDISP_ERR_INVALID_ARG;   // grid.y / grid.z of the pre-pass
    dedisp_status sst = scratch_reserve(plan, &plan->d_planes, &plan->planes_bytes, need, s);
    if (sst != DEDISP_OK || reserve_only) return sst;
    const int sms = plan->sm_count;
    sst = scratch_acquire(plan, s);
    if (sst != DEDISP_OK) return sst;

    if (plan->poison >= 0 && range.prepass) DEDISP_CUDA_TRY(plan, cudaMemsetAsync(plan->d_planes, plan->poison, plan->planes_bytes, s));
    if (plan->timing) cudaEventRecord(plan->ev[0], s);
    if (range.prepass && tscrunch == 1)
        DEDISP_CUDA_TRY(plan, launch_planes(C::NB, in, in_beam_stride, row_stride, plan->nchans, nbeams,
                                            plan->d_planes, (int)pitch, G.nchans_pad, s));
    else if (range.prepass)
        DEDISP_CUDA_TRY(plan, launch_planes_tscrunch(in_nbits, tscrunch, C::NB, in, in_beam_stride, row_stride,
                                                     plan->nchans, nbeams, plan->d_planes, (int)pitch,
                                                     G.nchans_pad, s));
    if (plan->timing) {
        cudaEventRecord(plan->ev[1], s);
        cudaEventRecord(plan->ev[2], s);
    }
    BitsliceParams P;
    P.planes = plan->d_planes;
    P.check_errors = plan->d_check_errors;
    P.inject_fault = plan->inject_fault;
    P.scratch_words = plan->planes_bytes / 4;
    P.ndm = plan->ndm;
    P.vinfo = nullptr;
    P.vlist = nullptr;
    P.vrows = 0;
    const BitsliceTables &T = plan->tab[G.tab];
    P.ws = T.d_ws;
    P.rel = T.d_rel;
    P.order = T.d_order;
    P.out = (uint8_t *)out;
    P.out_beam_stride = out_beam_stride;
    P.beam_pitch_words = beam_pitch;
    P.nsamps_out = nsamps_out;
    P.row_pitch = (int)pitch;
    P.nchans_pad = G.nchans_pad;
    P.ngroups = range.g_count > 0 ? range.g_count : G.ngroups;
    P.g_begin = range.g_begin;
    P.ntiles = (int)ntiles;
    P.nbeams = nbeams;
    // planes that fit L2 (126 MB) are re-read from it in any order; larger ones (8-bit wideband:
    // 750 MB) are walked tile-major inside blocks of gblock groups: gblock^2 ~ SMs x tile words x
    // groups / (max_delay / 32) balances the tiles in flight against the delay spread of a block
    P.gblock = 1;
    if (beam_pitch * 4 > (size_t)64 << 20) {
        const double spread = (double)(plan->max_delay >> 5) + 1.0;
        int gb = (int)std::sqrt((double)sms * C::TILE_WORDS * G.ngroups / spread);
        P.gblock = gb < 1 ? 1 : gb > P.ngroups ? P.ngroups : gb;
    }
    P.vec_ok = ((uintptr_t)out % 16 == 0) && (nsamps_out % 4 == 0) &&
               (nbeams == 1 || out_beam_stride % 16 == 0);
    const long long nitems = (long long)nbeams * P.ngroups * ntiles;
    const int grid = (int)(nitems < sms ? nitems : sms);
    // channel blocks: a block's largest possible sum must fit the NP counter planes; later blocks add to
    // the uint32 partial sums in out (float32 output: converted by the last block)
    const long long per_chan = (long long)tscrunch * ((1ll << in_nbits) - 1);
    long long cblk = (((1ll << C::NP) - 1) / per_chan) / CH_PAD * CH_PAD;
    if (cblk < CH_PAD) return DEDISP_ERR_INVALID_ARG;
    if (cblk > G.nchans_pad) cblk = G.nchans_pad;
    for (long long c0 = 0; c0 < G.nchans_pad; c0 += cblk) {
        const long long c1 = c0 + cblk < G.nchans_pad ? c0 + cblk : G.nchans_pad;
        P.chunk0 = (int)(c0 / C::CH);
        P.nchunks = (int)((c1 - c0) / C::CH);
        P.accumulate = c0 > 0;
        const bool f32 = out_f32 && c1 == G.nchans_pad;
        cudaError_t e;
        if (G.win_words == C::WIN_S)
            e = f32 ? launch_one<C, C::WIN_S, true>(P, grid, s, plan->device) : launch_one<C, C::WIN_S, false>(P, grid, s, plan->device);
        else
            e = f32 ? launch_one<C, C::WIN_L, true>(P, grid, s, plan->device) : launch_one<C, C::WIN_L, false>(P, grid, s, plan->device);
        DEDISP_CUDA_TRY(plan, e);
    }
    if (plan->timing) {
        cudaEventRecord(plan->ev[3], s);
        plan->timing_valid = true;
        plan->timing_has_prepass = true;
    }
    return scratch_release(plan, s);
}

// cuTensorMapEncodeTiled through the runtime's driver entry point (no link against libcuda)
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
inline EncodeTiledFn encode_tiled_fn()
{
    static std::atomic<EncodeTiledFn> fn{nullptr};
    EncodeTiledFn f = fn.load(std::memory_order_acquire);
    if (!f) {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn.store(f = (EncodeTiledFn)p, std::memory_order_release);
    }
    return f;
}

// Pair rows (pair_rows.cu): RAWNB-bit planes -> one (RAWNB+1)-plane row per (channel pair, delay difference) ->
// the tiled kernel over nchans/2 virtual channels (geometry C).  Same DM groups, tiles and row pitch as the
// plain geometry of the sample width.
template <class C, int RAWNB>
dedisp_status execute_pairs(dedisp_plan plan, const PairTables &T, int nbeams, long long nsamps_out,
                            const uint8_t *in, size_t row_stride, size_t in_beam_stride, void *out,
                            size_t out_beam_stride, int out_f32, cudaStream_t s, const BitsliceRange &range,
                            bool reserve_only)
{
    static_assert(C::NB == RAWNB + 1, "a pair sum has one more plane than a sample");
    const BitsliceGeom &G = plan->geom[geom_index(RAWNB)];
    const long long ntiles = (nsamps_out + C::TILE_SAMPS - 1) / C::TILE_SAMPS;
    const long long pitch =
        (((long long)(plan->max_delay >> 5) + ntiles * C::TILE_WORDS + C::WIN_S + 4) + 3) & ~3ll;
    if (ntiles > 0x7fffffff / C::TILE_WORDS || pitch > 0x7fffffff || nbeams > 65535) return DEDISP_ERR_INVALID_ARG;
    const size_t raw_beam = (size_t)G.nchans_pad * RAWNB * (size_t)pitch;
    const size_t rows_beam = (size_t)T.nrows * C::NB * (size_t)pitch;
    if ((unsigned long long)nbeams * T.nrows * C::NB > 0x7fffffffull) return DEDISP_ERR_INVALID_ARG;
    const size_t need_raw = raw_beam * (size_t)nbeams * 4, need_rows = rows_beam * (size_t)nbeams * 4;
    if (G.nchans_pad > 65535) return DEDISP_ERR_INVALID_ARG;   // grid.y of the unpack pre-pass
    dedisp_status sst = scratch_reserve(plan, &plan->d_planes, &plan->planes_bytes, need_raw, s);
    if (sst == DEDISP_OK) sst = scratch_reserve(plan, &plan->d_pair_rows, &plan->pair_rows_bytes, need_rows, s);
    if (sst != DEDISP_OK || reserve_only) return sst;
    const int sms = plan->sm_count;
    sst = scratch_acquire(plan, s);
    if (sst != DEDISP_OK) return sst;
    if (plan->poison >= 0 && range.prepass) {
        DEDISP_CUDA_TRY(plan, cudaMemsetAsync(plan->d_planes, plan->poison, plan->planes_bytes, s));
        DEDISP_CUDA_TRY(plan, cudaMemsetAsync(plan->d_pair_rows, plan->poison, plan->pair_rows_bytes, s));
    }
    if (plan->timing) cudaEventRecord(plan->ev[0], s);
    if (range.prepass) {
        DEDISP_CUDA_TRY(plan, launch_planes(RAWNB, in, in_beam_stride, row_stride, plan->nchans, nbeams,
                                            plan->d_planes, (int)pitch, G.nchans_pad, s));
        DEDISP_CUDA_TRY(plan, launch_pair_rows(T, RAWNB, plan->d_planes, raw_beam, G.nchans_pad, plan->d_pair_rows,
                                               rows_beam, (int)pitch, nbeams, s));
    }
    if (plan->timing) {
        cudaEventRecord(plan->ev[1], s);
        cudaEventRecord(plan->ev[2], s);
    }
    // the rows as a 2-D tensor [nbeams * nrows * NB lines][pitch words]; a box = the NB plane lines of one row x
    // one window (words outside the tensor read as zero: variant v starts vskew(v) words early)
    // (encoded once and kept in the plan: re-encoded only when the scratch pointer, the pitch or the line count change)
    TensorMapCache &tc = plan->tmap[RAWNB == 2 ? 0 : RAWNB == 4 ? 1 : 2];
    const unsigned long long lines = (unsigned long long)nbeams * T.nrows * C::NB;
    if (!tc.valid || tc.base != (void *)plan->d_pair_rows || tc.pitch != pitch || tc.lines != lines) {
        EncodeTiledFn enc = encode_tiled_fn();
        if (!enc) return DEDISP_ERR_CUDA;
        const cuuint64_t dims[2] = {(cuuint64_t)pitch, (cuuint64_t)lines};
        const cuuint64_t strides[1] = {(cuuint64_t)pitch * 4};
        const cuuint32_t box[2] = {(cuuint32_t)C::template plane_words<C::WIN_S>(), (cuuint32_t)C::NB};
        const cuuint32_t estr[2] = {1, 1};
        static_assert(sizeof(CUtensorMap) == sizeof(tc.map), "tensor map storage");
        if (enc(reinterpret_cast<CUtensorMap *>(tc.map), CU_TENSOR_MAP_DATA_TYPE_UINT32, 2, plan->d_pair_rows, dims,
                strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
            return DEDISP_ERR_CUDA;
        tc.valid = true;
        tc.base = plan->d_pair_rows;
        tc.pitch = pitch;
        tc.lines = lines;
    }
    const CUtensorMap &tm = *reinterpret_cast<const CUtensorMap *>(tc.map);
    BitsliceParams P;
    P.planes = plan->d_pair_rows;
    P.check_errors = plan->d_check_errors;
    P.inject_fault = plan->inject_fault;
    P.scratch_words = plan->pair_rows_bytes / 4;
    P.ndm = plan->ndm;
    P.vrows = T.nrows;
    P.ws = T.d_ws;
    P.rel = T.d_rel;
    P.vinfo = T.d_vinfo;
    P.vlist = nullptr;
    P.order = plan->tab[G.tab].d_order;
    P.out = (uint8_t *)out;
    P.out_beam_stride = out_beam_stride;
    P.beam_pitch_words = rows_beam;
    P.nsamps_out = nsamps_out;
    P.row_pitch = (int)pitch;
    P.nchans_pad = T.npairs_pad;
    P.ngroups = range.g_count > 0 ? range.g_count : G.ngroups;
    P.g_begin = range.g_begin;
    P.ntiles = (int)ntiles;
    P.nbeams = nbeams;
    // rows beyond L2: tile-major inside blocks of gblock groups, as in execute_cfg
    P.gblock = 1;
    if (rows_beam * 4 > (size_t)64 << 20 && RAWNB == 8) {
        const double spread = (double)(plan->max_delay >> 5) + 1.0;
        int gb = (int)std::sqrt((double)sms * C::TILE_WORDS * G.ngroups / spread);
        P.gblock = gb < 1 ? 1 : gb > P.ngroups ? P.ngroups : gb;
    }
    P.vec_ok = ((uintptr_t)out % 16 == 0) && (nsamps_out % 4 == 0) &&
               (nbeams == 1 || out_beam_stride % 16 == 0);
    const long long nitems = (long long)nbeams * P.ngroups * ntiles;
    const int grid = (int)(nitems < sms ? nitems : sms);
    // channel blocks as in execute_cfg: a pair sum is at most 2 (2^RAWNB - 1)
    long long cblk = (((1ll << C::NP) - 1) / (2 * ((1ll << RAWNB) - 1))) / CH_PAD * CH_PAD;
    if (cblk < CH_PAD) return DEDISP_ERR_INVALID_ARG;
    if (cblk > T.npairs_pad) cblk = T.npairs_pad;
    for (long long c0 = 0; c0 < T.npairs_pad; c0 += cblk) {
        const long long c1 = c0 + cblk < T.npairs_pad ? c0 + cblk : T.npairs_pad;
        P.chunk0 = (int)(c0 / C::CH);
        P.nchunks = (int)((c1 - c0) / C::CH);
        P.accumulate = c0 > 0;
        const bool f32 = out_f32 && c1 == T.npairs_pad;
        const cudaError_t e = f32 ? launch_one<C, C::WIN_S, true>(P, grid, s, plan->device, &tm)
                                  : launch_one<C, C::WIN_S, false>(P, grid, s, plan->device, &tm);
        DEDISP_CUDA_TRY(plan, e);
    }
    if (plan->timing) {
        cudaEventRecord(plan->ev[3], s);
        plan->timing_valid = true;
        plan->timing_has_prepass = true;
    }
    return scratch_release(plan, s);
}

// Quad rows (quad_rows.cu): RAWNB-bit planes -> one (RAWNB+2)-plane row per (channel quad, triple of delay
// differences) -> the tiled kernel over nchans/4 virtual channels (geometry C).  Same DM groups and tiles as the plain
// geometry of the sample width.
template <class C, int RAWNB>
dedisp_status execute_quads(dedisp_plan plan, const QuadTables &T, int nbeams, long long nsamps_out,
                            const uint8_t *in, size_t row_stride, size_t in_beam_stride, void *out,
                            size_t out_beam_stride, int out_f32, cudaStream_t s, const BitsliceRange &range,
                            bool reserve_only)
{
    static_assert(C::NB == RAWNB + 2, "a sum of four samples has two more planes than a sample");
    const BitsliceGeom &G = plan->geom[geom_index(RAWNB)];
    const long long ntiles = (nsamps_out + C::TILE_SAMPS - 1) / C::TILE_SAMPS;
    const long long pitch =
        (((long long)(plan->max_delay >> 5) + ntiles * C::TILE_WORDS + C::WIN_S + 4) + 3) & ~3ll;
    if (ntiles > 0x7fffffff / C::TILE_WORDS || pitch > 0x7fffffff || nbeams > 65535) return DEDISP_ERR_INVALID_ARG;
    const size_t raw_beam = (size_t)G.nchans_pad * RAWNB * (size_t)pitch;
    const size_t rows_beam = (size_t)T.nrows * C::NB * (size_t)pitch;
    if ((unsigned long long)nbeams * T.nrows * C::NB > 0x7fffffffull) return DEDISP_ERR_INVALID_ARG;
    const size_t need_raw = raw_beam * (size_t)nbeams * 4, need_rows = rows_beam * (size_t)nbeams * 4;
    if (G.nchans_pad > 65535) return DEDISP_ERR_INVALID_ARG;   // grid.y of the unpack pre-pass
    dedisp_status sst = scratch_reserve(plan, &plan->d_planes, &plan->planes_bytes, need_raw, s);
    if (sst == DEDISP_OK) sst = scratch_reserve(plan, &plan->d_pair_rows, &plan->pair_rows_bytes, need_rows, s);
    if (sst != DEDISP_OK || reserve_only) return sst;
    const int sms = plan->sm_count;
    sst = scratch_acquire(plan, s);
    if (sst != DEDISP_OK) return sst;
    if (plan->poison >= 0 && range.prepass) {
        DEDISP_CUDA_TRY(plan, cudaMemsetAsync(plan->d_planes, plan->poison, plan->planes_bytes, s));
        DEDISP_CUDA_TRY(plan, cudaMemsetAsync(plan->d_pair_rows, plan->poison, plan->pair_rows_bytes, s));
    }
    if (plan->timing) cudaEventRecord(plan->ev[0], s);
    if (range.prepass) {
        DEDISP_CUDA_TRY(plan, launch_planes(RAWNB, in, in_beam_stride, row_stride, plan->nchans, nbeams,
                                            plan->d_planes, (int)pitch, G.nchans_pad, s));
        DEDISP_CUDA_TRY(plan, launch_quad_rows(T, RAWNB, plan->d_planes, raw_beam, G.nchans_pad, plan->d_pair_rows,
                                               rows_beam, (int)pitch, nbeams, s));
    }
    if (plan->timing) {
        cudaEventRecord(plan->ev[1], s);
        cudaEventRecord(plan->ev[2], s);
    }
    // the rows as a 2-D tensor [nbeams * nrows * NB lines][pitch words]; a box = the NB plane lines of one row x
    // one window (words outside the tensor read as zero: a variant's box may start before its row or end after it)
    // (encoded once and kept in the plan: re-encoded only when the scratch pointer, the pitch or the line count change)
    TensorMapCache &tc = plan->tmap[3];
    const unsigned long long lines = (unsigned long long)nbeams * T.nrows * C::NB;
    if (!tc.valid || tc.base != (void *)plan->d_pair_rows || tc.pitch != pitch || tc.lines != lines) {
        EncodeTiledFn enc = encode_tiled_fn();
        if (!enc) return DEDISP_ERR_CUDA;
        const cuuint64_t dims[2] = {(cuuint64_t)pitch, (cuuint64_t)lines};
        const cuuint64_t strides[1] = {(cuuint64_t)pitch * 4};
        const cuuint32_t box[2] = {(cuuint32_t)C::template plane_words<C::WIN_S>(), (cuuint32_t)C::NB};
        const cuuint32_t estr[2] = {1, 1};
        static_assert(sizeof(CUtensorMap) == sizeof(tc.map), "tensor map storage");
        if (enc(reinterpret_cast<CUtensorMap *>(tc.map), CU_TENSOR_MAP_DATA_TYPE_UINT32, 2, plan->d_pair_rows, dims,
                strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
            return DEDISP_ERR_CUDA;
        tc.valid = true;
        tc.base = plan->d_pair_rows;
        tc.pitch = pitch;
        tc.lines = lines;
    }
    const CUtensorMap &tm = *reinterpret_cast<const CUtensorMap *>(tc.map);
    BitsliceParams P;
    P.planes = plan->d_pair_rows;
    P.check_errors = plan->d_check_errors;
    P.inject_fault = plan->inject_fault;
    P.scratch_words = plan->pair_rows_bytes / 4;
    P.ndm = plan->ndm;
    P.vrows = T.nrows;
    P.ws = T.d_ws;
    P.rel = T.d_rel;
    P.vinfo = nullptr;
    P.vlist = T.d_vlist;
    P.order = plan->tab[G.tab].d_order;
    P.out = (uint8_t *)out;
    P.out_beam_stride = out_beam_stride;
    P.beam_pitch_words = rows_beam;
    P.nsamps_out = nsamps_out;
    P.row_pitch = (int)pitch;
    P.nchans_pad = T.nquads_pad;
    P.ngroups = range.g_count > 0 ? range.g_count : G.ngroups;
    P.g_begin = range.g_begin;
    P.ntiles = (int)ntiles;
    P.nbeams = nbeams;
    // rows beyond L2: tile-major inside blocks of gblock groups, as in execute_cfg
    P.gblock = 1;
    if (rows_beam * 4 > (size_t)64 << 20) {
        const double spread = (double)(plan->max_delay >> 5) + 1.0;
        int gb = (int)std::sqrt((double)sms * C::TILE_WORDS * G.ngroups / spread);
        P.gblock = gb < 1 ? 1 : gb > P.ngroups ? P.ngroups : gb;
    }
    P.vec_ok = ((uintptr_t)out % 16 == 0) && (nsamps_out % 4 == 0) &&
               (nbeams == 1 || out_beam_stride % 16 == 0);
    const long long nitems = (long long)nbeams * P.ngroups * ntiles;
    const int grid = (int)(nitems < sms ? nitems : sms);
    // channel blocks as in execute_cfg: a quad sum is at most 4 (2^RAWNB - 1)
    long long cblk = (((1ll << C::NP) - 1) / (4 * ((1ll << RAWNB) - 1))) / CH_PAD * CH_PAD;
    if (cblk < CH_PAD) return DEDISP_ERR_INVALID_ARG;
    if (cblk > T.nquads_pad) cblk = T.nquads_pad;
    for (long long c0 = 0; c0 < T.nquads_pad; c0 += cblk) {
        const long long c1 = c0 + cblk < T.nquads_pad ? c0 + cblk : T.nquads_pad;
        P.chunk0 = (int)(c0 / C::CH);
        P.nchunks = (int)((c1 - c0) / C::CH);
        P.accumulate = c0 > 0;
        const bool f32 = out_f32 && c1 == T.nquads_pad;
        const cudaError_t e = f32 ? launch_one<C, C::WIN_S, true>(P, grid, s, plan->device, &tm)
                                  : launch_one<C, C::WIN_S, false>(P, grid, s, plan->device, &tm);
        DEDISP_CUDA_TRY(plan, e);
    }
    if (plan->timing) {
        cudaEventRecord(plan->ev[3], s);
        plan->timing_valid = true;
        plan->timing_has_prepass = true;
    }
    return scratch_release(plan, s);
}

}  // namespace bsk
