// bitslice_common.cuh -- geometry shared by the bit-plane pre-pass, the table
// builder and the tiled gather-sum kernel (all CUDA side; nothing here is used by
// the oracle).
//
// Data layout in HBM for the tiled kernel ("planes"): the packed filterbank is
// re-laid once per execute as bit planes,
//     planes[beam][c][p][word],   word w of plane p holds bit p of samples 32w .. 32w+31
//                                 of channel c (sample 32w+i in bit i),   p < nbits
// rows padded with zeros to `row_pitch` words (a multiple of 4 => every window the
// TMA bulk copies fetch is 16-byte aligned), channels padded with all-zero rows to a
// multiple of CH_PAD.  A (DM x time) tile of 32 trial DMs (one per lane) x TILE_WORDS
// words then needs, per channel and plane, one contiguous window of WIN words.
#pragma once
#include <stdint.h>

// tuning knobs of the 2-bit kernel (overridable with -D for A/B runs; defaults are
// the measured best, profiles/r1_*.md)
#ifndef BS_NW
#define BS_NW 15
#endif
#ifndef BS_W
#define BS_W 4
#endif
#ifndef BS_TREE_K
#define BS_TREE_K 4
#endif
#ifndef BS_NSTAGE
#define BS_NSTAGE 3
#endif
#ifndef BS_NSPLIT
#define BS_NSPLIT 1
#endif
#ifndef BS6_NSPLIT
#define BS6_NSPLIT 2
#endif

// ... and of the 8-bit kernel
#ifndef BS8_NW
#define BS8_NW 11
#endif
#ifndef BS8_W
#define BS8_W 4
#endif
#ifndef BS8_TREE_K
#define BS8_TREE_K 3
#endif
#ifndef BS8_NSTAGE
#define BS8_NSTAGE 3
#endif
#ifndef BS8_NSPLIT
#define BS8_NSPLIT 8      // round 2: one plane per tree -- with the carries chained across the subsets (add_chunk) more
#endif                    // subsets cost nothing and the 160-byte spill of NSPLIT = 2 is gone: wide8 on the plain kernel
                          // 57.1 -> 55.4 ms (NSPLIT 4: 55.6), profiles/r2_wide8.md
#ifndef BS8_WIN_S
#define BS8_WIN_S 80
#endif

// ... and of the 4-bit kernel
#ifndef BS4_NW
#define BS4_NW 11
#endif
#ifndef BS4_W
#define BS4_W 4
#endif
#ifndef BS4_TREE_K
#define BS4_TREE_K 3
#endif
#ifndef BS4_NSTAGE
#define BS4_NSTAGE 3
#endif
#ifndef BS4_NSPLIT
#define BS4_NSPLIT 1
#endif

namespace bs {
constexpr int LANES = 32;    // trial DMs per tile (one per lane)
constexpr int CH_PAD = 32;   // channels are padded to a multiple of this (>= every Cfg::CH)

// NB  input bit planes (= sample width)     NW  consumer warps per CTA
// W   32-sample words per thread per tile   K   adder-tree depth: 2^(K+1) channels per stage
// NP  accumulator bit planes (sums < 2^NP)  WIN_S / WIN_L  window words per (channel, plane)
// NSPLIT  the NB planes of a chunk go through NSPLIT adder trees of NB/NSPLIT planes each (a sample
//         is the sum of its bit fields): shorter-lived temporaries, so more warps fit the register file
// NV  variant windows staged per channel slot (1; 3 for the pair-sum rows, see Cfg3P below)
template <int NB_, int NW_, int W_, int K_, int NSTAGE_, int NP_, int WIN_S_, int WIN_L_, int NSPLIT_ = 1, int NV_ = 1>
struct Cfg {
    static constexpr int NB = NB_, NW = NW_, W = W_, K = K_, NSTAGE = NSTAGE_, NP = NP_, NV = NV_;
    static constexpr int NSPLIT = NSPLIT_, NBS = NB_ / NSPLIT_;
    // variant windows (NV > 1) are fetched as 2-D TMA boxes of NB plane lines x (WIN + VSKEW) words; the box of
    // an odd variant starts VSKEW = 16 words early, so its window sits 16 banks away from an even variant's: two
    // lanes of neighbouring variants collide on a bank only when their window offsets differ by exactly 16 words
    // (the offsets of a group span <= 17 words for the HTRU list, <= 24 for the 8-bit wideband one).  The variant
    // of a lane is NOT monotone in the lane -- delay[2p+1] - delay[2p] is a difference of two roundings and
    // toggles between neighbouring values from trial to trial -- so lanes of different variants interleave and a
    // small skew collides often: BS_VSKEW_UNIT=4 (variant v skewed by 4 v banks) measured 1.040 ms instead of
    // 0.935 ms on the HTRU gulp and 39.0 instead of 34.1 ms on the wideband (profiles/r2_wide8.md).
#ifdef BS_VSKEW_UNIT
    static constexpr int VSKEW = BS_VSKEW_UNIT * (NV_ - 1);
    static __host__ __device__ constexpr int vskew(int v) { return BS_VSKEW_UNIT * v; }
#else
    // up to 3 variants (pair rows): odd variants 16 banks away.  More (quad rows, NV = 7): no fixed skew -- every
    // variant of a (DM group, quad) has a box start of its own, placed by quad_prepare so that the lanes' words fall
    // into different banks (quad_rows.cu); VSKEW = 28 is the room the box leaves for that placement
    static constexpr int VSKEW = NV_ > 3 ? 28 : NV_ > 1 ? 16 : 0;
    static __host__ __device__ constexpr int vskew(int v)
    {
        return NV_ > 3 ? ((v & 1) * 16 + ((v >> 1) & 1) * 8 + ((v >> 2) & 1) * 4) : (v & 1) * VSKEW;
    }
#endif
    template <int WIN> static constexpr int plane_words() { return WIN + VSKEW; }
    template <int WIN> static constexpr int vslot_words()
    {
        return NV_ > 1 ? (NB_ * (WIN + VSKEW) + 31) / 32 * 32 : NB_ * WIN;   // boxes land 128-byte aligned
    }
    static constexpr int WIN_S = WIN_S_, WIN_L = WIN_L_;
    static constexpr int TILE_WORDS = NW * W;
    static constexpr int TILE_SAMPS = TILE_WORDS * 32;
    static constexpr int CH = 1 << (K + 1);          // channels per pipeline stage (one tree)
    static constexpr int NTHREADS = (NW + 1) * 32;   // + 1 producer warp
    static_assert(TILE_WORDS % 4 == 0, "tile starts must stay 16-byte aligned for the TMA bulk copies");
    static_assert(CH_PAD % CH == 0, "channel padding must cover whole stages");
    static_assert(NB + K + 1 <= NP, "tree carries must fit the accumulator");
};
// 2-bit samples: 15 x 4 words = 1920-sample tiles, 32-channel trees, sums < 4096
using Cfg2 = Cfg<2, BS_NW, BS_W, BS_TREE_K, BS_NSTAGE, 12, 96, 224, BS_NSPLIT>;
// 8-bit samples: 11 x 4 words = 1408-sample tiles, 16-channel trees run once per plane subset (round 1: NSPLIT = 2,
// the temporaries of a 4-plane tree leave room for 11 consumer warps at 168 registers; round 2: NSPLIT = 8), sums < 2^20
// (sweeps on B200, wide8, kernel ms.  One 8-plane tree, (NW,W,K,NSTAGE): (14,2,2,3) 81.6, (7,4,2,3) 75.0,
//  (6,4,2,3) 85.8, (12,2,3,3) 91.5, (10,2,3,3) 101.9, (7,4,3,3) 74.5 [ALU pipe 69 % busy: 2 warps per
//  sub-partition], (6,4,3,3) 84.9.  Split trees, (NSPLIT,NW,K,NSTAGE): (2,7,3,3) 73.7, (2,11,3,3) 60.7,
//  (2,11,3,2) 59.3, (2,11,2,3) 62.7, (4,11,3,3) 62.6, (4,15,3,3) 67.1, (8,15,3,3) 78.5, (8,11,3,3) 77.5;
//  window 80 instead of 128 words: 59.2 for 2, 3 or 4 stages)
using Cfg8 = Cfg<8, BS8_NW, BS8_W, BS8_TREE_K, BS8_NSTAGE, 20, BS8_WIN_S, 128, BS8_NSPLIT>;
// 1-bit samples (row f4): the packed row IS the bit plane; sums <= 4096 need 13 planes
using Cfg1 = Cfg<1, 15, 4, 4, 3, 13, 96, 224>;
// 4-bit samples (row f4): 11 x 4 words = 1408-sample tiles, 16-channel trees, sums < 2^16
// (sweep on B200, gulp at 4 bits: (NW,W,K,NSTAGE) = (10,4,2,3) 2.88 ms, (10,4,3,3) 2.62, (10,4,4,3) 2.53,
//  (11,4,3,3) 2.43, (9,4,3,3) 2.79, (12,3,2,3) 2.88, (14,2,3,3) 3.27)
using Cfg4 = Cfg<4, BS4_NW, BS4_W, BS4_TREE_K, BS4_NSTAGE, 16, 96, 224, BS4_NSPLIT>;

// 3-, 5- and 6-plane samples exist only as time-scrunched sums (row f4, reading R38:
// k samples of 1/2/4 bits added by the pre-pass): sums < 2^13 / 2^16 / 2^16
// (warps incl. the producer come in fours: the register file is per SM sub-partition)
#ifndef BS3_NW
#define BS3_NW 15
#endif
#ifndef BS3_TREE_K
#define BS3_TREE_K 3
#endif
#ifndef BS5_NW
#define BS5_NW 11
#endif
#ifndef BS5_TREE_K
#define BS5_TREE_K 3
#endif
#ifndef BS6_NW
#define BS6_NW 11
#endif
#ifndef BS6_TREE_K
#define BS6_TREE_K 3
#endif
using Cfg3 = Cfg<3, BS3_NW, 4, BS3_TREE_K, 3, 13, 96, 224>;
#ifndef BS5_NSPLIT
#define BS5_NSPLIT 5      // (one plane per tree: no spill; 8 x scrunched gulp 2.99 -> 2.90 ms)
#endif
using Cfg5 = Cfg<5, BS5_NW, 4, BS5_TREE_K, 3, 16, 96, 224, BS5_NSPLIT>;
using Cfg6 = Cfg<6, BS6_NW, 4, BS6_TREE_K, 3, 16, 96, 160, BS6_NSPLIT>;

// Pair sums: a virtual channel is the exact sum of two adjacent 2-bit
// channels, in[2p][t] + in[2p+1][t + delta], one 3-plane row per delay difference delta that occurs in the
// DM list; the trials of a group need at most NV = 3 consecutive differences (else the plan stays on Cfg2).
// Same tile as Cfg2 so that both paths share the DM groups and the row pitch.
// (sweeps on B200, HTRU gulp, step ms: (NW,W,K,NSTAGE) = (15,4,3,3) 1.03, (15,4,3,2) 1.06 [1.05 at the time],
//  (15,4,2,4) 1.13, (15,4,2,6) 1.14, (12,5,3,3) 1.13 [13 warps: 4 on one sub-partition, 128 registers, spills],
//  (10,6,3,3) 1.14, (20,3,3,3) 1.18 [80 registers, spills]; 16 consumers and no producer warp: 1.17)
#ifndef BS3P_NW
#define BS3P_NW 15
#endif
#ifndef BS3P_W
#define BS3P_W 4
#endif
#ifndef BS3P_TREE_K
#define BS3P_TREE_K 3
#endif
#ifndef BS3P_NSTAGE
#define BS3P_NSTAGE 3
#endif
using Cfg3P = Cfg<3, BS3P_NW, BS3P_W, BS3P_TREE_K, BS3P_NSTAGE, 13, 96, 96, 1, 3>;
// ... and of two adjacent 8-bit channels: 9-plane rows, three 3-plane adder trees per chunk of 8 pairs, same
// tile as Cfg8, sums < 2^20 (2048 pairs x 510); a stage is 82 KB, so the ring has two
#ifndef BS9P_NW
#define BS9P_NW 11
#endif
#ifndef BS9P_TREE_K
#define BS9P_TREE_K 2
#endif
#ifndef BS9P_NSTAGE
#define BS9P_NSTAGE 2
#endif
#ifndef BS9P_NSPLIT
#define BS9P_NSPLIT 3
#endif
// ... and of two adjacent 4-bit channels (row f4): 5-plane rows, same tile as Cfg4, sums < 2^16 (2048 pairs x
// 30); 16 pairs per stage make a stage 110 KB, so the ring has two (sweep on B200, gulp at 4 bits, step ms:
// (K,NSTAGE) = (3,2) 1.74, (2,3) 1.83, (2,4) 1.84)
#ifndef BS5P_NW
#define BS5P_NW 11
#endif
#ifndef BS5P_TREE_K
#define BS5P_TREE_K 3
#endif
#ifndef BS5P_NSTAGE
#define BS5P_NSTAGE 2
#endif
#ifndef BS5P_NSPLIT
#define BS5P_NSPLIT 5     // (one plane per tree: the 36-44 byte spill is gone; gulp at 4 bits, kernel 1.567 -> 1.512 ms)
#endif
using Cfg5P = Cfg<5, BS5P_NW, 4, BS5P_TREE_K, BS5P_NSTAGE, 16, 96, 96, BS5P_NSPLIT, 3>;
#ifndef BS9P_W
#define BS9P_W 4
#endif
#ifndef BS9P_WIN
#define BS9P_WIN BS8_WIN_S
#endif
using Cfg9P = Cfg<9, BS9P_NW, BS9P_W, BS9P_TREE_K, BS9P_NSTAGE, 20, BS9P_WIN, BS9P_WIN, BS9P_NSPLIT, 3>;

// Quad rows (quad_rows.cu): a virtual channel is the exact sum of FOUR adjacent 8-bit channels at fixed delay
// differences (d1, d2, d3) to the first of them, one 10-plane row per difference triple that occurs in the DM list;
// the trials of a group use at most NV = 7 distinct triples of a quad (else the plan stays on the pair rows).  Four
// quads (16 channels) per stage, one plane per adder tree; window 72 + 28 words of skew per plane line.
#ifndef BS10Q_NW
#define BS10Q_NW 11
#endif
using Cfg10Q = Cfg<10, BS10Q_NW, 4, 1, 2, 20, 72, 72, 10, 7>;

constexpr int NGEOM = 9;                                   // geometries are indexed by plane count 1..8
constexpr int geom_index(int nplanes) { return nplanes; }
// planes needed for the block sums of k samples of nbits bits, rounded up to a built geometry (0: none)
inline int tscrunch_planes(int nbits, int k)
{
    const long long maxv = (long long)k * ((1 << nbits) - 1);
    int nb = 1;
    while ((1ll << nb) <= maxv) ++nb;
    return nb <= 6 ? nb : nb <= 8 ? 8 : 0;
}
}  // namespace bs

struct BitsliceParams {
    const uint32_t *planes;    // [nbeams][nchans_pad][NB][row_pitch]
    const int32_t *ws;         // [ngroups][nchans_pad] window start word (multiple of 4)
    const uint32_t *rel;       // [ngroups][nchans_pad][32] (byte offset in window << 16) | bit shift
    const int32_t *order;      // [ngroups*32] output row of each lane, -1 = padding lane
    uint8_t *out;
    size_t out_beam_stride;    // bytes
    size_t beam_pitch_words;   // words between beams in planes
    long long nsamps_out;
    int row_pitch;             // words
    int nchans_pad;
    int ngroups;               // DM groups this launch covers ...
    int g_begin;               // ... starting at this group of the sorted list
    int ntiles;                // time tiles per (beam, group)
    int nbeams;
    int chunk0, nchunks;       // channel chunks [chunk0, chunk0 + nchunks) of Cfg::CH channels are summed ...
    int accumulate;            // ... and added to what out already holds (channel blocks, sums >= 2^NP)
    int gblock;                // work-item order: blocks of gblock DM groups, inside a block tile-major
    int vec_ok;                // output rows are 16-byte aligned: 128-bit stores allowed
    // pair rows (Cfg::NV > 1): planes = [nbeams][nrows][NB][row_pitch], a channel slot of group g stages rows
    // (vinfo & 0x0fffffff) .. + (vinfo >> 28) of it; rel carries the lane's variant in its byte offset
    const uint32_t *vinfo;     // [ngroups][nchans_pad]
    int vrows;                 // rows per beam
    // quad rows (Cfg::NV > 3): the rows a slot stages are listed explicitly, vlist[(group * nchans_pad + slot) * NV + v]
    // = (row of variant v or -1, first word of its box for tile 0): every variant has a window start of its own, placed
    // so that the lanes of the group fall into different shared-memory banks (quad_rows.cu)
    const int2 *vlist;
    // self-checks (library built with -DDEDISP_CHECKS; see dedisp_debug_check_errors): failure counters in device
    // memory and the extent of the scratch the producer may read
    unsigned long long *check_errors;   // [DEDISP_NCHECK] or nullptr
    unsigned long long scratch_words;   // words in `planes`
    int ndm;
    int inject_fault;                   // dedisp_debug_inject_fault: 1 = stamp a wrong tag on one ring stage
};
// what the self-checks count (index into check_errors)
enum {
    CHK_TOTAL = 0,          // all failures
    CHK_LDS_RANGE = 1,      // a consumer's shared-memory reads would leave the stage's data area
    CHK_STAGE_TAG = 2,      // a consumer found another (work item, chunk) in the stage than the one it waited for
    CHK_TMA_SRC = 3,        // a bulk copy / tensor box would read outside the scratch (beyond the designed zero-fill margin)
    CHK_OUT_RANGE = 4,      // the epilogue's output row or sample range is outside out
    CHK_PREPASS = 5,        // a pre-pass thread would write outside its row
    DEDISP_NCHECK = 8
};
