// dedisp_internal.h -- private declarations shared by the translation units of
// libdedisp_b200.so.  Not part of the ABI (see include/dedisp.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <vector>

#include "dedisp.h"

// Geometry of the bit-sliced tiled kernel (bitslice_kernel.cu).
struct BitsliceGeom {
    bool usable = false;     // plan can be served by the bit-sliced kernel
    int nbits = 0;           // geometry was derived for this sample width
    int nchans_pad = 0;      // channels padded to a multiple of the chunk size
    int ndm_pad = 0;         // DM trials padded to a multiple of 32 (lanes)
    int ngroups = 0;         // ndm_pad / 32
    int win_words = 0;       // smem words per (channel, plane) window
    int nplanes_acc = 0;     // accumulator bit planes
    int tab = 0;             // which table set (dedisp_plan_s::tab) the geometry reads
};

// Tables of the tiled kernel for one grouping of the sorted trial DMs: groups of 32 lanes of which
// the first dms_per_group hold trials (32 unless the DM steps are so coarse that the delays of 32
// neighbouring trials would not fit a tile window; then 16, 8, ... and the other lanes idle).
struct BitsliceTables {
    uint32_t *d_rel = nullptr;    // [ngroups][nchans_pad][32] packed (byte offset<<16 | shift)
    int32_t *d_ws = nullptr;      // [ngroups][nchans_pad] window start word
    int32_t *d_order = nullptr;   // [ngroups*32] trial index of each lane, -1 = idle lane
    int ngroups = 0;
    int dms_per_group = 0;
    int max_off = 0;              // largest (delay >> 5) - window start over the table, words
};

// Tables of the pair-row path (pair_rows.cu): virtual channel p = channels 2p and 2p+1 summed at a fixed
// delay difference; one 3-plane row per (pair, difference) that occurs in the DM list.
struct PairTables {
    uint32_t *d_rel = nullptr;      // [ngroups][npairs_pad][32] ((variant slot + window offset) bytes << 16) | shift
    int32_t *d_ws = nullptr;        // [ngroups][npairs_pad] window start word (of channel 2p)
    uint32_t *d_vinfo = nullptr;    // [ngroups][npairs_pad] first row | (rows - 1) << 28
    int32_t *d_pair_row0 = nullptr; // [npairs_pad] first row of each pair ...
    int32_t *d_pair_dlo = nullptr;  // [npairs_pad] ... its delay difference (rows of a pair: consecutive differences)
    int32_t *d_pair_cnt = nullptr;  // [npairs_pad] rows of the pair
    int nrows = 0;
    int npairs_pad = 0;
    bool usable = false;
};

struct dedisp_plan_s {
    int nchans = 0;
    double dt = 0, f_top = 0, df = 0;
    int ndm = 0;
    std::vector<double> dms;
    int device = 0;
    int32_t *d_delay = nullptr;   // [nchans][ndm]
    int max_delay = -1;
    dedisp_kernel want = DEDISP_KERNEL_AUTO;
    int last_kernel = 0;
    int bitslice_kind = DEDISP_KERNEL_BITSLICE;   // which tiled variant the last bitslice_execute ran
    int last_cuda_error = 0;
    // bit-sliced path: tables built by set_dm_list, scratch grown lazily by execute
    BitsliceGeom geom[9];         // [bit planes per sample]: 1, 2, 4, 8 = packed widths; 3, 5, 6 = time-scrunched sums
    BitsliceTables tab[2];        // [0] for the 96/224-word windows, [1] for the narrower 8-/6-plane windows
    uint32_t *d_planes = nullptr; // bit-plane copy of the input
    size_t planes_bytes = 0;
    PairTables pairs;             // pair-row path, 2-bit samples (Cfg3P, DM groups of tab[0])
    PairTables pairs4;            // pair-row path, 4-bit samples (Cfg5P, DM groups of tab[0])
    PairTables pairs8;            // pair-row path, 8-bit samples (Cfg9P, DM groups of tab[1])
    uint32_t *d_pair_rows = nullptr;
    size_t pair_rows_bytes = 0;
    // dedisp_execute_host staging
    void *d_in_stage = nullptr;
    size_t in_stage_bytes = 0;
    void *d_out_stage = nullptr;
    size_t out_stage_bytes = 0;
    cudaStream_t host_stream = nullptr;
    cudaStream_t copy_stream = nullptr;   // device->host copies of finished DM ranges / beams
    cudaEvent_t chunk_ev[16] = {};
    bool order_identity = false;          // trial DMs were given in ascending order: sorted lane = output row
    // optional per-kernel timing: ev[0..1] around the pre-pass, ev[2..3] around the main kernel
    bool timing = false;
    bool timing_valid = false;
    bool timing_has_prepass = false;
    cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
};

extern unsigned long long g_launch_count;

#define DEDISP_CUDA_TRY(plan, expr)                         \
    do {                                                    \
        cudaError_t e_ = (expr);                            \
        if (e_ != cudaSuccess) {                            \
            if (plan) (plan)->last_cuda_error = (int)e_;    \
            return DEDISP_ERR_CUDA;                         \
        }                                                   \
    } while (0)

// delay_table.cu
cudaError_t launch_delay_table(int nchans, double dt, double f_top, double df, const double *d_dms,
                               int ndm, int32_t *d_delay, int *d_max_delay, int *d_overflow,
                               cudaStream_t s);

// direct_kernel.cu
cudaError_t launch_direct(const int32_t *d_delay, int nchans, int ndm, long long nsamps_out,
                          const uint8_t *in, size_t row_stride, size_t in_beam_stride, int nbits,
                          void *out, size_t out_beam_stride, int out_f32, int nbeams,
                          cudaStream_t s);

// bitslice_prepare.cu / bitslice_kernel.cu
cudaError_t launch_planes(int nbits, const uint8_t *in, size_t in_beam_stride, size_t row_stride,
                          int nchans, int nbeams, uint32_t *planes, int row_pitch, int nchans_pad,
                          cudaStream_t s);
// time-scrunch pre-passes (row f4): block sums of k samples -> `nplanes` bit planes / one byte per sum
cudaError_t launch_planes_tscrunch(int nbits, int k, int nplanes, const uint8_t *in, size_t in_beam_stride,
                                   size_t row_stride, int nchans, int nbeams, uint32_t *planes,
                                   int row_pitch, int nchans_pad, cudaStream_t s);
cudaError_t launch_tscrunch_bytes(int nbits, int k, const uint8_t *in, size_t in_beam_stride, size_t row_stride,
                                  int nchans, int nbeams, long long nsamps_scr, uint8_t *out, cudaStream_t s);
dedisp_status bitslice_prepare(dedisp_plan plan);   // called at the end of set_dm_list
void bitslice_release(dedisp_plan plan);
// returns DEDISP_OK, or DEDISP_ERR_INVALID_ARG when the plan cannot use this kernel
// tscrunch = 1: plain; 2/4/8/16: the pre-pass sums blocks of tscrunch samples (row_stride = fine row)
// range (optional): only DM groups [g_begin, g_begin + g_count) of the sorted list; prepass = false
// re-uses the bit planes a previous call on this plan left in the scratch (same input, same shape)
struct BitsliceRange {
    int g_begin = 0;
    int g_count = 0;      // 0 = all groups
    bool prepass = true;
};
dedisp_status bitslice_execute(dedisp_plan plan, int nbeams, long long nsamps_out,
                               const uint8_t *in, size_t row_stride, size_t in_beam_stride,
                               int nbits, int tscrunch, void *out, size_t out_beam_stride, int out_f32,
                               cudaStream_t s, const BitsliceRange *range = nullptr);
// pair_rows.cu
dedisp_status pair_prepare(dedisp_plan plan);       // after bitslice_prepare; leaves pairs.usable
void pair_release(dedisp_plan plan);
cudaError_t launch_pair_rows(const PairTables &T, int raw_nbits, const uint32_t *raw, size_t raw_beam_pitch, int nchans_pad,
                             uint32_t *rows, size_t rows_beam_pitch, int row_pitch, int nbeams, cudaStream_t s);
// DM groups of the plan's bit-sliced geometry for this sample width, or 0 if the kernel cannot serve it
int bitslice_ngroups(dedisp_plan plan, int nbits);
