// dedisp_internal.h -- private declarations shared by the translation units of
// libdedisp_b200.so.  Not part of the ABI (see include/dedisp.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>
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

// Tables of the quad-row path (quad_rows.cu): virtual channel q = channels 4q .. 4q+3 summed at fixed delay differences
// (d1, d2, d3) to channel 4q; one (nbits + 2)-plane row per (quad, triple) that occurs in the DM list.
struct QuadTables {
    uint32_t *d_rel = nullptr;      // [ngroups][nquads_pad][32] ((variant slot + word in the variant's box) bytes << 16) | shift
    int32_t *d_ws = nullptr;        // [ngroups][nquads_pad] window start word (of channel 4q; kept for the checks)
    int2 *d_vlist = nullptr;        // [ngroups][nquads_pad][NV] (row of each variant the group uses or -1, box start word)
    int32_t *d_row0 = nullptr;      // [nquads_pad + 1] first row of each quad (rows of a quad: triples in ascending order)
    int32_t *d_trip = nullptr;      // [nrows][4] (d1, d2, d3, 0) of each row
    int nrows = 0;
    int nquads_pad = 0;
    bool usable = false;
};

// The encoded 2-D tensor map of the pair rows (cuTensorMapEncodeTiled), kept until the scratch moves or the shape changes.
struct TensorMapCache {
    alignas(64) unsigned char map[128] = {};
    bool valid = false;
    void *base = nullptr;
    long long pitch = 0;
    unsigned long long lines = 0;
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
    QuadTables quads8;            // quad-row path, 8-bit samples (Cfg10Q, DM groups of tab[1])
    TensorMapCache tmap[4];       // pair rows of 2-, 4- and 8-bit samples; quad rows of 8-bit samples
    // diagnostics (dedisp_debug_set_poison / dedisp_debug_check_errors)
    int poison = -1;                               // >= 0: every execute first fills the scratch with this byte
    int inject_fault = 0;                          // -DDEDISP_CHECKS builds: a deliberate fault the checks must count
    unsigned long long *d_check_errors = nullptr;  // [DEDISP_NCHECK] failure counters of a -DDEDISP_CHECKS build
    int sm_count = 0;             // multiprocessors of `device` (set_dm_list)
    // ordering of the plan-owned scratch between executes on different streams: the stream and an event after the
    // last kernels that touched it (scratch_acquire / scratch_release, dedisp_api.cu)
    cudaStream_t scratch_stream = nullptr;
    cudaEvent_t scratch_ev = nullptr;
    bool scratch_ev_valid = false;
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

extern std::atomic<unsigned long long> g_launch_count;

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
                               cudaStream_t s, const BitsliceRange *range = nullptr, bool reserve_only = false);

// One call of the tiled kernel in a given geometry; the geometries are instantiated by one translation unit each
// (bitslice_inst_*.cu) so that they compile in parallel.
struct BitsliceCall {
    dedisp_plan plan;
    const BitsliceGeom *G;
    int nbeams;
    long long nsamps_out;
    const uint8_t *in;
    size_t row_stride, in_beam_stride;
    int in_nbits, tscrunch;
    void *out;
    size_t out_beam_stride;
    int out_f32;
    cudaStream_t s;
    BitsliceRange range;
    bool reserve_only;        // grow the scratch for this call and return (dedisp_reserve)
};
dedisp_status bitslice_run_cfg1(const BitsliceCall &c);
dedisp_status bitslice_run_cfg2(const BitsliceCall &c);
dedisp_status bitslice_run_cfg3(const BitsliceCall &c);
dedisp_status bitslice_run_cfg4(const BitsliceCall &c);
dedisp_status bitslice_run_cfg5(const BitsliceCall &c);
dedisp_status bitslice_run_cfg6(const BitsliceCall &c);
dedisp_status bitslice_run_cfg8(const BitsliceCall &c);
dedisp_status bitslice_run_pairs2(const BitsliceCall &c);
dedisp_status bitslice_run_pairs4(const BitsliceCall &c);
dedisp_status bitslice_run_pairs8(const BitsliceCall &c);
dedisp_status bitslice_run_quads8(const BitsliceCall &c);

// Plan-owned scratch (dedisp_api.cu).  reserve: grow *ptr to `need` bytes (cudaFree + cudaMalloc: synchronises the
// device, so nothing in flight still reads the old buffer; refused with DEDISP_ERR_CUDA while `s` is being captured
// into a graph -- call dedisp_reserve before capturing).  acquire / release bracket the kernels of one execute:
// an execute on another stream than the previous one first waits for the event the previous one recorded.
dedisp_status scratch_reserve_bytes(dedisp_plan plan, void **ptr, size_t *have, size_t need, cudaStream_t s);
template <class T>
inline dedisp_status scratch_reserve(dedisp_plan plan, T **ptr, size_t *have, size_t need, cudaStream_t s)
{
    return scratch_reserve_bytes(plan, reinterpret_cast<void **>(ptr), have, need, s);
}
dedisp_status scratch_acquire(dedisp_plan plan, cudaStream_t s);
dedisp_status scratch_release(dedisp_plan plan, cudaStream_t s);
// pair_rows.cu
dedisp_status pair_prepare(dedisp_plan plan);       // after bitslice_prepare; leaves pairs.usable
void pair_release(dedisp_plan plan);
cudaError_t launch_pair_rows(const PairTables &T, int raw_nbits, const uint32_t *raw, size_t raw_beam_pitch, int nchans_pad,
                             uint32_t *rows, size_t rows_beam_pitch, int row_pitch, int nbeams, cudaStream_t s);
// quad_rows.cu
dedisp_status quad_prepare(dedisp_plan plan);       // after pair_prepare; leaves quads8.usable
void quad_release(dedisp_plan plan);
cudaError_t launch_quad_rows(const QuadTables &T, int raw_nbits, const uint32_t *raw, size_t raw_beam_pitch, int nchans_pad,
                             uint32_t *rows, size_t rows_beam_pitch, int row_pitch, int nbeams, cudaStream_t s);
// DM groups of the plan's bit-sliced geometry for this sample width, or 0 if the kernel cannot serve it
int bitslice_ngroups(dedisp_plan plan, int nbits);

// matched_filter.cu: the dense pass (z and / or RMS + block maxima) or, with sparse_list, the re-computation of listed
// blocks into a compact z (dedisp_search_events, peak_finding.cu)
dedisp_status mf_run(const void *x_dev, dedisp_out_dtype x_dtype, long long nrows, long long nsamps, int radius,
                     const int *widths_host, int nwidths, unsigned int x_max, float *z_dev, float *rms_dev,
                     int *blockmax_dev, void *workspace_dev, size_t workspace_bytes, void *cuda_stream,
                     const int2 *sparse_list, const int *sparse_count, float *zc, long long max_blocks);
// matched_filter_warp.cu: the same passes by the warp-autonomous kernel (no dense z), and its segment length
dedisp_status mf_warp_run(const void *x_dev, dedisp_out_dtype x_dtype, long long nrows, long long nsamps, int radius,
                          const int *widths_host, int nwidths, unsigned int x_max, float *z_dev, float *rms_dev,
                          int *blockmax_dev, void *workspace_dev, size_t workspace_bytes, void *cuda_stream,
                          const int2 *sparse_list, const int *sparse_count, float *zc, long long max_blocks);
long long mf_warp_segment(long long nrows, long long nsamps);
size_t mf_warp_workspace_bytes(long long nrows, long long nsamps, int nwidths);   // partial sums + per-row prefix sums
