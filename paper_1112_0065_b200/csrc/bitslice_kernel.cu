// bitslice_kernel.cu -- dispatch of the tiled gather-sum (kernel C, bitslice_kernel.cuh): which geometry serves a call
// (sample width, time scrunch, pair rows or plain planes).  The kernel itself is instantiated per geometry in
// bitslice_inst_*.cu.
//
//   out[d][t] = sum_c in[c][t + delay[c][d]]       (BASELINE.json:north_star)
#include "bitslice_common.cuh"
#include "dedisp_internal.h"

using namespace bs;

// AUTO takes the pair rows when the tiles saved outweigh building the rows once per execute: measured on B200
// (HTRU gulp, profiles/r1j_pairs.md) a tile of a DM group is 6.2 us / 35 cheaper per 512 pairs and a row costs
// 12 bytes per word at 3.7 TB/s, i.e. break-even near ngroups * npairs = 0.6 * nrows; and when the rows of all
// beams stay below PAIRS_MAX_BYTES of scratch.
#ifndef PAIRS_GAIN_NUM
#define PAIRS_GAIN_NUM 4       // pairs when PAIRS_GAIN_DEN * ngroups * npairs >= PAIRS_GAIN_NUM * nrows
#endif
#ifndef PAIRS_GAIN_DEN
#define PAIRS_GAIN_DEN 5
#endif
#ifndef PAIRS8_AUTO
#define PAIRS8_AUTO 1          // 8-bit pair rows (wide8: 59.9 -> 41.2 ms per step; the same break-even holds)
#endif
#ifndef QUADS8_AUTO
#define QUADS8_AUTO 1
#endif
#ifndef PAIRS_MAX_BYTES
#define PAIRS_MAX_BYTES (24ull << 30)
#endif


dedisp_status bitslice_execute(dedisp_plan plan, int nbeams, long long nsamps_out,
                               const uint8_t *in, size_t row_stride, size_t in_beam_stride,
                               int nbits, int tscrunch, void *out, size_t out_beam_stride, int out_f32,
                               cudaStream_t s, const BitsliceRange *range, bool reserve_only)
{
    const BitsliceRange full;
    const BitsliceRange &rg = range ? *range : full;
    // bit planes per (block-summed) sample; a scrunch factor the pre-pass does not build is not served here
    const bool pow2 = tscrunch == 2 || tscrunch == 4 || tscrunch == 8 || tscrunch == 16;
    if (tscrunch != 1 && !(pow2 && nbits * tscrunch <= 32)) return DEDISP_ERR_INVALID_ARG;
    const int np = tscrunch == 1 ? nbits : tscrunch_planes(nbits, tscrunch);
    if (np < 1 || np >= NGEOM) return DEDISP_ERR_INVALID_ARG;
    const BitsliceGeom &G = plan->geom[geom_index(np)];
    // (sums beyond the counter planes are served in channel blocks as long as 32 channels fit)
    const long long per_chan = (long long)tscrunch * ((1ll << nbits) - 1);
    if (!G.usable || CH_PAD * per_chan >= (1ll << G.nplanes_acc)) return DEDISP_ERR_INVALID_ARG;
    if (rg.g_begin < 0 || rg.g_count < 0 || rg.g_begin + rg.g_count > G.ngroups) return DEDISP_ERR_INVALID_ARG;
    // pair rows: 2-, 4- and 8-bit samples at full time resolution.  AUTO takes them when the DM list is long enough for
    // the rows (built once per execute, ~max_delay/2 + nchans/2 of them) to pay for themselves.
    const PairTables &PT = nbits == 8 ? plan->pairs8 : nbits == 4 ? plan->pairs4 : plan->pairs;
    const BitsliceCall call = {plan, &G, nbeams, nsamps_out, in, row_stride, in_beam_stride, nbits, tscrunch, out,
                               out_beam_stride, out_f32, s, rg, reserve_only};
    const bool pairs_fit = (nbits == 2 || nbits == 4 || nbits == 8) && tscrunch == 1 && PT.usable;
    if (plan->want == DEDISP_KERNEL_PAIRS && !pairs_fit) return DEDISP_ERR_INVALID_ARG;
    // quad rows (8-bit samples at full time resolution): the step after the pair rows.  AUTO takes them when a (DM
    // group, quad) amortises its share of the rows -- measured on B200 (profiles/r2_wide8.md) a quad slot of a DM group
    // is ~240 ns x SMs cheaper than its two pair slots and a row costs ~60 ns to build, break-even near 4 rows per
    // (group, quad): taken at <= 3 -- and the rows of all beams stay below PAIRS_MAX_BYTES of scratch.
    const QuadTables &QT = plan->quads8;
    const bool quads_fit = nbits == 8 && tscrunch == 1 && QT.usable;
    if (plan->want == DEDISP_KERNEL_QUADS && !quads_fit) return DEDISP_ERR_INVALID_ARG;
    bool quads_pay = false;
    if (quads_fit && plan->want == DEDISP_KERNEL_AUTO && (rg.prepass || plan->bitslice_kind == DEDISP_KERNEL_QUADS)) {
        const long long ntiles = (nsamps_out + Cfg10Q::TILE_SAMPS - 1) / Cfg10Q::TILE_SAMPS;
        const unsigned long long bytes = (unsigned long long)QT.nrows * Cfg10Q::NB * 4ull * (unsigned long long)nbeams *
                                         (unsigned long long)((plan->max_delay >> 5) + ntiles * Cfg10Q::TILE_WORDS + 128);
        quads_pay = (long long)QT.nrows <= 3ll * G.ngroups * QT.nquads_pad && bytes <= PAIRS_MAX_BYTES && QUADS8_AUTO;
    }
    if (quads_fit && (plan->want == DEDISP_KERNEL_QUADS || quads_pay)) {
        plan->bitslice_kind = DEDISP_KERNEL_QUADS;
        const dedisp_status st = bitslice_run_quads8(call);
        if (st != DEDISP_ERR_ALLOC || plan->want != DEDISP_KERNEL_AUTO) return st;      // (else: pair rows, then planes)
    }
    bool pairs_pay = false;
    // (a DM-group range that continues an execute -- no pre-pass of its own -- stays on what the first range ran)
    if (pairs_fit && plan->want == DEDISP_KERNEL_AUTO && (rg.prepass || plan->bitslice_kind == DEDISP_KERNEL_PAIRS)) {
        const int tile_words = nbits == 8 ? Cfg9P::TILE_WORDS : nbits == 4 ? Cfg5P::TILE_WORDS : Cfg3P::TILE_WORDS;
        const long long ntiles = (nsamps_out + 32 * tile_words - 1) / (32 * tile_words);
        const unsigned long long bytes = (unsigned long long)PT.nrows * (nbits + 1) * 4ull * (unsigned long long)nbeams *
                                         (unsigned long long)((plan->max_delay >> 5) + ntiles * tile_words + 128);
        pairs_pay = (long long)PAIRS_GAIN_DEN * G.ngroups * PT.npairs_pad >= (long long)PAIRS_GAIN_NUM * PT.nrows &&
                    bytes <= PAIRS_MAX_BYTES && (nbits != 8 || PAIRS8_AUTO);
    }
    if (pairs_fit && (plan->want == DEDISP_KERNEL_PAIRS || pairs_pay)) {
        plan->bitslice_kind = DEDISP_KERNEL_PAIRS;
        const dedisp_status st = nbits == 4 ? bitslice_run_pairs4(call) : nbits == 8 ? bitslice_run_pairs8(call)
                                                                                     : bitslice_run_pairs2(call);
        // AUTO never fails where the plain tiled kernel would not: when the scratch for the rows cannot be
        // allocated (nothing has been enqueued at that point) the call is served from the planes instead
        if (st != DEDISP_ERR_ALLOC || plan->want != DEDISP_KERNEL_AUTO) return st;
    }
    plan->bitslice_kind = DEDISP_KERNEL_BITSLICE;
    switch (np) {
        case 1: return bitslice_run_cfg1(call);
        case 2: return bitslice_run_cfg2(call);
        case 3: return bitslice_run_cfg3(call);
        case 4: return bitslice_run_cfg4(call);
        case 5: return bitslice_run_cfg5(call);
        case 6: return bitslice_run_cfg6(call);
        default: return bitslice_run_cfg8(call);
    }
}

int bitslice_ngroups(dedisp_plan plan, int nbits)
{
    if (nbits < 1 || nbits >= NGEOM) return 0;
    const BitsliceGeom &G = plan->geom[geom_index(nbits)];
    // (the host path maps a range of groups to a range of output rows: needs 32 trials in every group)
    return (G.usable && plan->tab[G.tab].dms_per_group == 32 &&
            CH_PAD * ((1ll << nbits) - 1) < (1ll << G.nplanes_acc)) ? G.ngroups : 0;
}
