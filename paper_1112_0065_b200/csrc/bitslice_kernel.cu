// bitslice_kernel.cu -- kernel C: the tiled gather-sum (north_star subsystem (c), (d)).
//
//   out[d][t] = sum_c in[c][t + delay[c][d]]       (BASELINE.json:north_star)
//
// B200 design:
//   * a work item = (beam, group of 32 trial DMs, tile of 2048 output samples);
//     persistent CTAs (one per SM) walk the item list;
//   * lane  = trial DM, warp = 4 consecutive 32-sample words, 16 consumer warps;
//   * one producer warp stages, per 16-channel chunk, the window of bit-plane words
//     the tile needs with 1-D TMA bulk copies (cp.async.bulk + mbarrier tx counts)
//     into a 4-deep shared-memory ring, so neighbouring DMs reuse one staged window;
//   * consumers never unpack to integers: a sample stays 2 bit planes, is aligned
//     with one funnel shift per plane-word and is added with carry-save adders
//     (2 LOP3 per full adder) into a 12-plane bit-sliced counter held in registers
//     -- 32 additions per instruction, ~0.2 ALU ops per (channel, DM, sample);
//   * the counter is un-sliced once per tile and written as uint32 / float32.
#include "bitslice_common.cuh"
#include "dedisp_internal.h"

using namespace bs;

namespace {

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

// full adder on 32 independent bit positions: acc <- acc ^ x ^ y, returns majority(acc, x, y)
__device__ __forceinline__ uint32_t full_add(uint32_t &acc, uint32_t x, uint32_t y)
{
    uint32_t carry, sum;
    asm("lop3.b32 %0, %1, %2, %3, 0xE8;" : "=r"(carry) : "r"(acc), "r"(x), "r"(y));
    asm("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(sum) : "r"(acc), "r"(x), "r"(y));
    acc = sum;
    return carry;
}

template <int WIN>
struct Stage {
    static constexpr int CPITCH = 2 * WIN * 4;          // bytes per channel: plane 0 then plane 1
    static constexpr int DATA_BYTES = CH * CPITCH;
    static constexpr int REL_BYTES = CH * LANES * 4;
    static constexpr int BYTES = DATA_BYTES + REL_BYTES;
};

// Load the W+1 words of both planes of channel C that this thread's 4 output words
// need, and align them to the output time axis (one funnel shift per plane-word).
template <int C, int WIN>
__device__ __forceinline__ void load_aligned(const uint8_t *tb, const uint32_t *relp,
                                             uint32_t (&a)[W], uint32_t (&b)[W])
{
    const uint32_t r = relp[C * LANES];
    const uint32_t *wp = reinterpret_cast<const uint32_t *>(tb + (r >> 16)) + C * (2 * WIN);
    uint32_t w0[W + 1], w1[W + 1];
#pragma unroll
    for (int j = 0; j <= W; ++j) {
        w0[j] = wp[j];
        w1[j] = wp[WIN + j];
    }
#pragma unroll
    for (int j = 0; j < W; ++j) {
        a[j] = __funnelshift_r(w0[j], w0[j + 1], r);   // shift amount = r & 31
        b[j] = __funnelshift_r(w1[j], w1[j + 1], r);
    }
}

// Tree<K> adds 2^(K+1) channels (C0 ...) into the counter planes 0..K+1 and hands
// back one carry word of weight 2^(K+1) (u) and one of weight 2^(K+2) (v).
template <int K, int C0, int WIN>
struct Tree {
    template <int NP>
    static __device__ __forceinline__ void run(uint32_t (&A)[NP][W], const uint8_t *tb,
                                               const uint32_t *relp, uint32_t (&u)[W],
                                               uint32_t (&v)[W])
    {
        uint32_t u1[W], v1[W], u2[W], v2[W];
        Tree<K - 1, C0, WIN>::run(A, tb, relp, u1, v1);
        Tree<K - 1, C0 + (1 << K), WIN>::run(A, tb, relp, u2, v2);
#pragma unroll
        for (int j = 0; j < W; ++j) {
            u[j] = full_add(A[K][j], u1[j], u2[j]);
            v[j] = full_add(A[K + 1][j], v1[j], v2[j]);
        }
    }
};
template <int C0, int WIN>
struct Tree<0, C0, WIN> {
    template <int NP>
    static __device__ __forceinline__ void run(uint32_t (&A)[NP][W], const uint8_t *tb,
                                               const uint32_t *relp, uint32_t (&u)[W],
                                               uint32_t (&v)[W])
    {
        uint32_t a0[W], b0[W], a1[W], b1[W];
        load_aligned<C0, WIN>(tb, relp, a0, b0);
        load_aligned<C0 + 1, WIN>(tb, relp, a1, b1);
#pragma unroll
        for (int j = 0; j < W; ++j) {
            u[j] = full_add(A[0][j], a0[j], a1[j]);   // bit 0 of both channels
            v[j] = full_add(A[1][j], b0[j], b1[j]);   // bit 1 of both channels
        }
    }
};


template <int WIN, int NP, bool F32>
__global__ void __launch_bounds__(NTHREADS, 1) bitslice_dedisperse(const BitsliceParams P, int vec_ok)
{
    extern __shared__ __align__(128) uint8_t smem[];
    using S = Stage<WIN>;
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem + NSTAGE * S::BYTES);
    const uint32_t full0 = smem_u32(bars), empty0 = smem_u32(bars + NSTAGE);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int s = 0; s < NSTAGE; ++s) {
            mbar_init(full0 + 8 * s, 1);
            mbar_init(empty0 + 8 * s, NW);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const int nchunks = P.nchans_pad / CH;
    const long long nitems = (long long)P.nbeams * P.ngroups * P.ntiles;
    int stage = 0;
    uint32_t phase = 0;

    if (warp == NW) {
        // ---------------- producer warp: TMA bulk copies into the ring ----------------
        for (long long item = blockIdx.x; item < nitems; item += gridDim.x) {
            const int tile = (int)(item % P.ntiles);
            const int g = (int)((item / P.ntiles) % P.ngroups);
            const int beam = (int)(item / ((long long)P.ntiles * P.ngroups));
            const uint32_t *pl = P.planes + (size_t)beam * P.beam_pitch_words + (size_t)tile * TILE_WORDS;
            const size_t grow = (size_t)g * P.nchans_pad;
            for (int chunk = 0; chunk < nchunks; ++chunk) {
                mbar_wait(empty0 + 8 * stage, phase ^ 1);
                const uint32_t sb = smem_u32(smem) + stage * S::BYTES;
                const uint32_t fb = full0 + 8 * stage;
                if (lane == 0) mbar_expect_tx(fb, S::BYTES);
                __syncwarp();
                // one copy per (channel, plane) of the chunk: CH * 2 copies spread over the lanes
#pragma unroll
                for (int i = lane; i < CH * 2; i += 32) {
                    const int c = chunk * CH + (i >> 1), pidx = i & 1;
                    const uint32_t *src = pl + ((size_t)c * 2 + pidx) * P.row_pitch + P.ws[grow + c];
                    bulk_g2s(sb + i * (WIN * 4), src, WIN * 4, fb);
                }
                if (lane == 0)
                    bulk_g2s(sb + S::DATA_BYTES, P.rel + (grow + (size_t)chunk * CH) * LANES,
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
            uint32_t u[W], v[W];
            Tree<TREE_K, 0, WIN>::run(A, tb, relp, u, v);
            // fold the two carry words (weights 2^(K+1), 2^(K+2)) into the upper planes
#pragma unroll
            for (int j = 0; j < W; ++j) {
                uint32_t c = u[j];
                uint32_t t = A[TREE_K + 1][j] & c;
                A[TREE_K + 1][j] ^= c;
                c = full_add(A[TREE_K + 2][j], t, v[j]);
#pragma unroll
                for (int p = TREE_K + 3; p < NP - 1; ++p) {
                    t = A[p][j] & c;
                    A[p][j] ^= c;
                    c = t;
                }
                A[NP - 1][j] ^= c;
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(empty0 + 8 * stage);
            if (++stage == NSTAGE) { stage = 0; phase ^= 1; }
        }

        // ---------------- epilogue: un-slice the counter, convert, store ----------------
        const int tile = (int)(item % P.ntiles);
        const int g = (int)((item / P.ntiles) % P.ngroups);
        const int beam = (int)(item / ((long long)P.ntiles * P.ngroups));
        const int d = P.order[g * LANES + lane];
        uint8_t *orow = P.out + (size_t)beam * P.out_beam_stride +
                        (size_t)(d < 0 ? 0 : d) * (size_t)P.nsamps_out * 4;
#pragma unroll
        for (int j = 0; j < W; ++j) {
            const long long t0 = (long long)tile * TILE_SAMPS + (warp * W + j) * 32;
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                uint32_t lo = 0, hi = 0;
#pragma unroll
                for (int p = 0; p < NP; ++p) {
                    const uint32_t n = (A[p][j] >> (4 * q)) & 0xFu;
                    // spread the 4 bits of n to bit (p & 7) of the 4 bytes
                    const int pp = p & 7;
                    const uint32_t s = (n * (0x00204081u << pp)) & (0x01010101u << pp);
                    if (p < 8) lo |= s; else hi |= s;
                }
                uint32_t o[4];
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    o[k] = __byte_perm(lo, hi, 0x40 + 0x11 * k) & 0xFFFFu;
                    if (F32) o[k] = __float_as_uint(__uint_as_float(o[k] | 0x4B000000u) - 8388608.0f);
                }
                const long long t = t0 + 4 * q;
                if (d >= 0) {
                    if (vec_ok && t + 3 < P.nsamps_out) {
                        *reinterpret_cast<uint4 *>(orow + (size_t)t * 4) = make_uint4(o[0], o[1], o[2], o[3]);
                    } else {
#pragma unroll
                        for (int k = 0; k < 4; ++k)
                            if (t + k < P.nsamps_out)
                                *reinterpret_cast<uint32_t *>(orow + (size_t)(t + k) * 4) = o[k];
                    }
                }
            }
#pragma unroll
            for (int p = 0; p < NP; ++p) A[p][j] = 0;
        }
    }
}

template <int WIN, int NP, bool F32>
cudaError_t launch_one(const BitsliceParams &P, int vec_ok, int grid, cudaStream_t s)
{
    constexpr int SMEM = NSTAGE * Stage<WIN>::BYTES + 2 * NSTAGE * 8;
    static bool attr_done = false;
    if (!attr_done) {
        cudaError_t e = cudaFuncSetAttribute(bitslice_dedisperse<WIN, NP, F32>,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM);
        if (e != cudaSuccess) return e;
        attr_done = true;
    }
    bitslice_dedisperse<WIN, NP, F32><<<grid, NTHREADS, SMEM, s>>>(P, vec_ok);
    ++g_launch_count;
    return cudaGetLastError();
}

}  // namespace

dedisp_status bitslice_execute(dedisp_plan plan, int nbeams, long long nsamps_out,
                               const uint8_t *in, size_t row_stride, size_t in_beam_stride,
                               int nbits, void *out, size_t out_beam_stride, int out_f32,
                               cudaStream_t s)
{
    if (nbits != 2) return DEDISP_ERR_INVALID_ARG;
    const BitsliceGeom &G = plan->geom[0];
    if (!G.usable) return DEDISP_ERR_INVALID_ARG;
    const long long ntiles = (nsamps_out + TILE_SAMPS - 1) / TILE_SAMPS;
    const long long pitch = (((long long)(plan->max_delay >> 5) + ntiles * TILE_WORDS + G.win_words + 4) + 3) & ~3ll;
    if (ntiles > 0x7fffffff / TILE_WORDS || pitch > 0x7fffffff) return DEDISP_ERR_INVALID_ARG;
    const size_t beam_pitch = (size_t)G.nchans_pad * 2 * (size_t)pitch;
    const size_t need = beam_pitch * (size_t)nbeams * 4;
    if (plan->planes_bytes < need) {
        cudaFree(plan->d_planes);
        plan->d_planes = nullptr;
        plan->planes_bytes = 0;
        if (cudaMalloc(&plan->d_planes, need) != cudaSuccess) {
            cudaGetLastError();
            return DEDISP_ERR_ALLOC;
        }
        plan->planes_bytes = need;
    }
    int sms = 0;
    DEDISP_CUDA_TRY(plan, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, plan->device));

    if (plan->timing) cudaEventRecord(plan->ev[0], s);
    DEDISP_CUDA_TRY(plan, launch_planes2(in, in_beam_stride, row_stride, plan->nchans, nbeams,
                                         plan->d_planes, (int)pitch, G.nchans_pad, s));
    if (plan->timing) {
        cudaEventRecord(plan->ev[1], s);
        cudaEventRecord(plan->ev[2], s);
    }
    BitsliceParams P;
    P.planes = plan->d_planes;
    P.ws = plan->d_ws[0];
    P.rel = plan->d_rel[0];
    P.order = plan->d_order;
    P.out = (uint8_t *)out;
    P.out_beam_stride = out_beam_stride;
    P.beam_pitch_words = beam_pitch;
    P.nsamps_out = nsamps_out;
    P.row_pitch = (int)pitch;
    P.nchans_pad = G.nchans_pad;
    P.ngroups = G.ngroups;
    P.ntiles = (int)ntiles;
    P.nbeams = nbeams;
    const long long nitems = (long long)nbeams * G.ngroups * ntiles;
    const int grid = (int)(nitems < sms ? nitems : sms);
    const int vec_ok = ((uintptr_t)out % 16 == 0) && (nsamps_out % 4 == 0) &&
                       (nbeams == 1 || out_beam_stride % 16 == 0);
    cudaError_t e;
    if (G.win_words == WIN_SMALL)
        e = out_f32 ? launch_one<WIN_SMALL, 12, true>(P, vec_ok, grid, s)
                    : launch_one<WIN_SMALL, 12, false>(P, vec_ok, grid, s);
    else
        e = out_f32 ? launch_one<WIN_LARGE, 12, true>(P, vec_ok, grid, s)
                    : launch_one<WIN_LARGE, 12, false>(P, vec_ok, grid, s);
    DEDISP_CUDA_TRY(plan, e);
    if (plan->timing) {
        cudaEventRecord(plan->ev[3], s);
        plan->timing_valid = true;
        plan->timing_has_prepass = true;
    }
    return DEDISP_OK;
}
