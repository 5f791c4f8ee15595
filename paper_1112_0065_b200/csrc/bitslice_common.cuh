// bitslice_common.cuh -- geometry shared by the bit-plane pre-pass, the table
// builder and the tiled gather-sum kernel (all CUDA side; nothing here is used by
// the oracle).
//
// Data layout in HBM for the tiled kernel ("planes"): the packed filterbank is
// re-laid once per execute as bit planes,
//     planes[beam][c][p][word],   word w of plane p holds bit p of samples 32w .. 32w+31
//                                 of channel c (sample 32w+i in bit i),
// rows padded with zeros to `row_pitch` words (a multiple of 4 => every window the
// TMA bulk copies fetch is 16-byte aligned), channels padded with all-zero rows to a
// multiple of CH.  A (DM x time) tile of 32 trial DMs (one per lane) x TILE_WORDS
// words then needs, per channel and plane, one contiguous window of WIN words.
#pragma once
#include <stdint.h>

// tuning knobs (overridable with -D for A/B runs; defaults are the measured best)
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

namespace bs {
constexpr int NW = BS_NW;               // consumer warps per CTA
constexpr int W = BS_W;                 // 32-sample words per thread per tile
constexpr int TILE_WORDS = NW * W;      // 60 words
constexpr int TILE_SAMPS = TILE_WORDS * 32;   // 1920 output samples per tile
constexpr int LANES = 32;               // trial DMs per tile (one per lane)
constexpr int TREE_K = BS_TREE_K;       // adder tree depth: 2^(K+1) channels per tree
constexpr int CH = 1 << (TREE_K + 1);   // channels per pipeline stage (one tree)
constexpr int NSTAGE = BS_NSTAGE;       // TMA ring depth
constexpr int NTHREADS = (NW + 1) * 32; // + 1 producer warp
constexpr int WIN_SMALL = 96;           // window words per (channel, plane): small DM steps
constexpr int WIN_LARGE = 224;          // large DM steps
static_assert(TILE_WORDS % 4 == 0, "tile starts must stay 16-byte aligned for the TMA bulk copies");
}  // namespace bs

struct BitsliceParams {
    const uint32_t *planes;    // [nbeams][nchans_pad][NPL][row_pitch]
    const int32_t *ws;         // [ngroups][nchans_pad] window start word (multiple of 4)
    const uint32_t *rel;       // [ngroups][nchans_pad][32] (byte offset in window << 16) | bit shift
    const int32_t *order;      // [ngroups*32] output row of each lane, -1 = padding lane
    uint8_t *out;
    size_t out_beam_stride;    // bytes
    size_t beam_pitch_words;   // words between beams in planes
    long long nsamps_out;
    int row_pitch;             // words
    int nchans_pad;
    int ngroups;
    int ntiles;                // time tiles per (beam, group)
    int nbeams;
};
