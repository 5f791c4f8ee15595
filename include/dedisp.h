/*
 * dedisp.h -- C ABI of libdedisp_b200: direct (brute-force) incoherent
 * dedispersion on one NVIDIA B200 (sm_100a).
 *
 * The operation (BASELINE.json:north_star; Sec. 2.2 "each dispersion
 * trial involves a complete integration over frequency channels"
 * Sec. 2.2 "the most common 'direct' dedispersion algorithm"):
 *
 *     out[d][t] = sum_{c=0}^{nchans-1} in[c][ t + delay[c][d] ]
 *     delay[c][d] = round( 4148.808 * DM_d * ( f_c^-2 - f_top^-2 ) / dt )
 *     f_c = f_top + c*df          (MHz; dt in seconds; DM in pc cm^-3)
 *
 * round() is to nearest, ties away from zero, on the IEEE double value of the
 * expression evaluated as ((4148.808*DM) * (1/(f_c*f_c) - 1/(f_top*f_top))) / dt
 * with one rounding per operation (no FMA contraction).
 *
 * Every step (delay table, unpack, gather-sum, output conversion) runs in CUDA
 * kernels.  There is no CPU fallback: without a usable CUDA device every call
 * that needs one returns DEDISP_ERR_CUDA.
 *
 * Layouts
 *   in   packed samples, channel-major: nchans rows, each row holds
 *        nsamps_in = nsamps_out + max_delay samples, time contiguous.
 *        2-bit: 4 samples per byte, LSB first: sample t of a row is
 *               (row[t>>2] >> (2*(t&3))) & 3.   8-bit: one unsigned byte per sample.
 *        1- and 4-bit (input-format variants): the same rule,
 *               sample t = bits [t*nbits, (t+1)*nbits) of the row as a little-endian bit string.
 *        Row stride is TIGHT: dedisp_get_in_row_stride_bytes() =
 *        ceil(nsamps_in*nbits/8) bytes; no alignment is required of the base
 *        pointer or of the rows.  Bits past the last sample of a row are never read
 *        as samples.
 *   out  [ndm][nsamps_out], t fastest, tight, uint32 or float32 (exact: every sum
 *        is < 2^24).  The base pointer must be 4-byte aligned.
 *   batch  in[beam][c][t], out[beam][d][t] with caller-given beam strides in bytes.
 *
 * Ownership: the plan and everything it allocates on the device belong to the
 * library (released by dedisp_destroy).  in/out buffers and the stream belong to
 * the caller.  Host arrays passed in are copied before the call returns.
 *
 * Threading: a plan is not thread-safe; distinct plans are independent (two host
 * threads may drive two plans concurrently; the library's only process-wide state, the
 * launch counter and the per-kernel attribute flags, is atomic).
 *
 * Streams and scratch: the execute calls only enqueue work on the caller's stream.  A plan
 * owns device scratch (bit planes, pair or quad rows) that every execute of that plan re-uses:
 * executes of ONE plan are therefore ordered -- a call on another stream than the plan's
 * previous call first waits (cudaStreamWaitEvent) for the event the previous call recorded
 * behind its kernels, so double-buffered callers stay correct but two executes of one plan
 * never overlap; use one plan per concurrent stream for overlap.  The scratch is grown on
 * demand inside execute with cudaFree + cudaMalloc (which synchronises the device);
 * dedisp_reserve sizes it ahead of time so that the steady state never allocates.  While a
 * stream is being captured into a CUDA graph the scratch cannot grow (execute returns
 * DEDISP_ERR_CUDA, last error cudaErrorStreamCaptureUnsupported): call dedisp_reserve before
 * capturing.  A captured graph holds the scratch pointers of its capture: it is invalidated
 * when a later, larger execute / dedisp_reserve, or dedisp_set_dm_list, re-allocates them.
 *
 * Reads of `in`: only bytes of the caller's rows are read -- the unpack pre-pass uses aligned
 * 128-bit loads for 16-byte blocks that lie inside [in, in + extent) and byte loads for the
 * partial first / last block of the buffer, so nothing before `in` or past the last row's end
 * is touched, whatever the alignment.
 *
 * Errors: every entry point returns a dedisp_status (or a value documented
 * below); nothing throws or aborts across the ABI.
 */
#ifndef DEDISP_B200_H
#define DEDISP_B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dedisp_plan_s *dedisp_plan; /* opaque, library-owned */

typedef enum {
    DEDISP_OK = 0,
    DEDISP_ERR_INVALID_ARG = 1,       /* null pointer, non-positive size, bad geometry */
    DEDISP_ERR_NO_DM_LIST = 2,        /* execute/getter before dedisp_set_dm_list */
    DEDISP_ERR_UNSUPPORTED_NBITS = 3, /* in_nbits not in {1, 2, 4, 8} */
    DEDISP_ERR_UNSUPPORTED_DTYPE = 4, /* out_dtype not U32/F32 */
    DEDISP_ERR_OVERFLOW = 5,          /* nchans*(2^nbits-1) >= 2^24, or a delay beyond int32 */
    DEDISP_ERR_ALLOC = 6,             /* host or device allocation failed */
    DEDISP_ERR_CUDA = 7,              /* CUDA runtime error; see dedisp_get_last_cuda_error */
    DEDISP_ERR_SCRATCH_LIMIT = 8      /* dedisp_execute_static: the problem needs more than the fixed static scratch */
} dedisp_status;

typedef enum { DEDISP_OUT_U32 = 0, DEDISP_OUT_F32 = 1 } dedisp_out_dtype;

/* Kernel selection (diagnostics and A/B evidence; default AUTO). */
typedef enum {
    DEDISP_KERNEL_AUTO = 0,     /* bit-sliced tiled kernel when the plan fits it, else DIRECT */
    DEDISP_KERNEL_DIRECT = 1,   /* one thread per output group, reads packed input from global */
    DEDISP_KERNEL_BITSLICE = 2, /* TMA-staged (DM x time) tiles, bit-plane carry-save adders */
    DEDISP_KERNEL_PAIRS = 3,    /* the same tiled kernel on pair rows: in[2p][t] + in[2p+1][t + delta] is formed
                                   once per delay difference delta of the DM list (nbits + 1 bit planes) and the tiles
                                   add nchans/2 such rows -- the identical integer sum, re-associated.  2-, 4-
                                   and 8-bit samples; AUTO picks it when the plan fits (see dedisp_get_last_kernel)
                                   and falls back to the plain tiled kernel when the scratch for the rows
                                   cannot be allocated (forced PAIRS then returns DEDISP_ERR_ALLOC);
                                   BITSLICE forces the plain tiled kernel */
    DEDISP_KERNEL_QUADS = 4     /* ... and on quad rows: the sum of FOUR adjacent channels formed once per triple of delay
                                   differences of the DM list (nbits + 2 planes), nchans/4 rows per output.  8-bit samples
                                   only; needs up to tens of GB of scratch for long DM lists (8-bit wideband config:
                                   20.3 GB); up to 4096 channels, >= 8 DM groups, <= 7 distinct triples per group and
                                   quad, else forced QUADS returns INVALID_ARG; AUTO takes it when it pays and fits,
                                   else pair rows, else planes */
} dedisp_kernel;

/* Create a plan for nchans channels, sample time dt_s (s), channel 0 at f_top_mhz,
 * channel spacing df_mhz (MHz, must be < 0 so that delays are >= 0).
 * host-only; rejects nchans < 1, dt <= 0, f_top <= 0, df >= 0,
 * f_top + (nchans-1)*df <= 0, non-finite values.  (north_star: dedisp_plan_create) */
dedisp_status dedisp_plan_create(dedisp_plan *plan, int nchans, double dt_s, double f_top_mhz,
                                 double df_mhz);

/* Copy ndm trial DMs (HOST pointer, doubles, any order, duplicates allowed; each
 * finite and >= 0) and build the delay table ON THE DEVICE (fp64, rule above).
 * May be called again to replace the list.  Synchronous.
 * (north_star: dedisp_set_dm_list, subsystem (a).) */
dedisp_status dedisp_set_dm_list(dedisp_plan plan, const double *dms_host, int ndm);

/* Dedisperse one beam.  in_dev/out_dev are DEVICE pointers (layouts above);
 * cuda_stream is a cudaStream_t passed as void* (NULL = legacy default stream).
 * Only enqueues work on the stream; does not synchronise.
 * (north_star: dedisp_execute, subsystems (b),(c).) */
dedisp_status dedisp_execute(dedisp_plan plan, long long nsamps_out, const void *in_dev,
                             int in_nbits, void *out_dev, dedisp_out_dtype out_dtype,
                             void *cuda_stream);

/* Same for nbeams independent beams in one batched launch (north_star subsystem (d),
 * BASELINE.json configs[4]; 13 beams: PAPER.md:18).  Beam b reads
 * in_dev + b*in_beam_stride_bytes and writes out_dev + b*out_beam_stride_bytes
 * (out stride a multiple of 4). */
dedisp_status dedisp_execute_batch(dedisp_plan plan, int nbeams, long long nsamps_out,
                                   const void *in_dev, size_t in_beam_stride_bytes, int in_nbits,
                                   void *out_dev, size_t out_beam_stride_bytes,
                                   dedisp_out_dtype out_dtype, void *cuda_stream);

/* Dedispersion at reduced time resolution ("time scrunching", SURVEY.md Sec. 8(f) row f4;
 * DESIGN.md reading R38 -- the paper only says that ~1200 trial DMs are searched).
 * Every input row is first summed in non-overlapping blocks of `tscrunch` samples (block 0 starts
 * at sample 0; raw sums, no division), and the block sums are dedispersed on the coarse grid:
 *
 *     s[c][u]   = sum_{j < tscrunch} in[c][tscrunch*u + j]
 *     out[d][t] = sum_c s[c][ t + delay[c][d] ]
 *
 * `plan` describes the COARSE grid: create it with dt_s = tscrunch * (the input's sample time);
 * delay[][] and max_delay are in coarse samples.  Each input row holds
 * tscrunch * (nsamps_out + max_delay) samples of in_nbits bits in a tight row of
 * dedisp_get_in_row_stride_bytes_tscrunch() bytes; out is [ndm][nsamps_out] as for dedisp_execute;
 * beams as in dedisp_execute_batch.  Requires tscrunch >= 1 and tscrunch*(2^in_nbits - 1) <= 255
 * (else DEDISP_ERR_INVALID_ARG) and nchans*tscrunch*(2^in_nbits - 1) < 2^24 (else
 * DEDISP_ERR_OVERFLOW).  tscrunch = 1 is dedisp_execute_batch.  Factors 2, 4, 8, 16 with
 * in_nbits*tscrunch <= 32 are summed inside the bit-plane pre-pass and run the bit-sliced kernel
 * on 2..6 (or 8) planes; any other factor is summed to bytes and served by the DIRECT kernel.
 * Only enqueues work on the stream. */
dedisp_status dedisp_execute_tscrunch(dedisp_plan plan, int tscrunch, int nbeams, long long nsamps_out,
                                      const void *in_dev, size_t in_beam_stride_bytes, int in_nbits,
                                      void *out_dev, size_t out_beam_stride_bytes,
                                      dedisp_out_dtype out_dtype, void *cuda_stream);
/* ceil(tscrunch * (nsamps_out + max_delay) * in_nbits / 8); 0 on error. */
size_t dedisp_get_in_row_stride_bytes_tscrunch(dedisp_plan plan, int tscrunch, long long nsamps_out,
                                               int in_nbits);

/* Grow the plan's scratch to what dedisp_execute_batch(plan, nbeams, nsamps_out, .., in_nbits, ..)
 * needs with the kernel selection in force (AUTO: quad or pair rows where they pay, else bit planes), so that
 * later executes of that size or smaller never allocate (see "Streams and scratch").  Synchronises
 * the device if it has to re-allocate.  Errors: INVALID_ARG, NO_DM_LIST, UNSUPPORTED_NBITS, ALLOC. */
dedisp_status dedisp_reserve(dedisp_plan plan, int nbeams, long long nsamps_out, int in_nbits);

/* dedisp_execute for callers that cannot call cudaMalloc (code under CUDA-graph capture, tight serving loops,
 * harnesses that forbid it): one beam through the plain tiled kernel (what DEDISP_KERNEL_BITSLICE runs: unpack
 * pre-pass -> bit planes -> TMA-staged gather-sum), with the bit planes in a file-scope device array of
 * DEDISP_STATIC_SCRATCH_BYTES (32 MiB) instead of the plan's cudaMalloc'ed scratch.  The call -- the first one
 * included -- calls no cudaMalloc / cudaFree and no allocating library routine; the first call on a device looks the
 * array's device address up (cudaGetSymbolAddress; CUDA loads modules lazily, so this is also when the driver
 * reserves the 32 MiB) and sets the kernel's shared-memory attribute, and a plan's first call outside a capture
 * creates the plan's ordering event: make one call outside a capture first.  Same arguments, layouts and result (bit for bit) as dedisp_execute; the current device
 * must be the one dedisp_set_dm_list ran on.
 *   Limit: the bit planes of the call, nchans_pad * in_nbits * row_pitch * 4 bytes (row_pitch ~ (nsamps_out +
 *   max_delay) / 32 + 200 words, nchans_pad = nchans rounded up to 32), must fit 32 MiB -- the HTRU gulp (1024 channels,
 *   2 bits, 65 536 + 20 476 samples: 23.3 MB) does, the 8-bit wideband config (750 MB) does not: DEDISP_ERR_SCRATCH_LIMIT.
 *   Plans the tiled kernel cannot serve return DEDISP_ERR_INVALID_ARG (there is no DIRECT fallback here).
 *   Cost: every GPU that loads the library holds the 32 MiB until the process exits; no pair rows (they need 373 MB for
 *   the gulp), so the gulp takes 1.20 ms instead of 1.04 ms.
 *   Sharing: the array is ONE per process and device, shared by all plans, streams and threads, and keeps the last
 *   call's contents (nothing needs clearing: the pre-pass rewrites every word a call reads).  Calls that overlap on the
 *   GPU race on it and give wrong sums: serialise them (one stream, or events).  Calls of one plan on different
 *   streams are ordered as for dedisp_execute. */
#define DEDISP_STATIC_SCRATCH_BYTES (32u << 20)
size_t dedisp_static_scratch_bytes(void);
dedisp_status dedisp_execute_static(dedisp_plan plan, long long nsamps_out, const void *in_dev, int in_nbits,
                                    void *out_dev, dedisp_out_dtype out_dtype, void *cuda_stream);

/* End-to-end convenience with HOST buffers (tight beam strides): copies the
 * packed input host->device, runs dedisp_execute_batch, copies the result back
 * and synchronises.  Device staging buffers, two streams and a few events are owned
 * and reused by the plan.  The result dominates the transfer time, so it leaves in
 * pieces while the kernel still runs on the rest: one beam at a time, or -- single
 * beam, trial DMs given in ascending order -- up to 8 ranges of DM groups (output rows).
 * Pinned host memory gives full PCIe rate and the overlap; pageable memory works too. */
dedisp_status dedisp_execute_host(dedisp_plan plan, int nbeams, long long nsamps_out,
                                  const void *in_host, int in_nbits, void *out_host,
                                  dedisp_out_dtype out_dtype);

/* Release the plan and all device memory it owns.  NULL is accepted. */
dedisp_status dedisp_destroy(dedisp_plan plan);

/* ---- getters (valid after dedisp_set_dm_list unless noted) ---- */

/* Largest entry of the delay table in samples, or -1 without a DM list. */
int dedisp_get_max_delay(dedisp_plan plan);
int dedisp_get_nchans(dedisp_plan plan); /* valid after create */
int dedisp_get_ndm(dedisp_plan plan);    /* 0 without a DM list */

/* ceil((nsamps_out + max_delay) * in_nbits / 8); 0 on error. */
size_t dedisp_get_in_row_stride_bytes(dedisp_plan plan, long long nsamps_out, int in_nbits);

/* Copy the device-built delay table to host_out[nchans][ndm] (int32, d fastest). */
dedisp_status dedisp_get_delay_table(dedisp_plan plan, int *host_out);

/* Force a kernel variant for subsequent executes (default DEDISP_KERNEL_AUTO).
 * Forcing BITSLICE, PAIRS or QUADS on a plan it cannot serve makes execute return INVALID_ARG. */
dedisp_status dedisp_set_kernel(dedisp_plan plan, dedisp_kernel which);
/* Variant the last execute on this plan used (DEDISP_KERNEL_DIRECT/BITSLICE/PAIRS/QUADS), 0 if none. */
int dedisp_get_last_kernel(dedisp_plan plan);

/* Per-kernel device timing (for the bench's roofline line).  When enabled, execute
 * records CUDA events on the caller's stream around the pre-pass (bit-plane unpack)
 * and around the dominant gather-sum kernel.  dedisp_get_last_kernel_ms waits for
 * the last execute's events and returns both durations in milliseconds
 * (prepass 0 when the DIRECT kernel ran). */
dedisp_status dedisp_set_timing(dedisp_plan plan, int enable);
dedisp_status dedisp_get_last_kernel_ms(dedisp_plan plan, float *prepass_ms, float *main_ms);

/* ---- downstream of dedispersion ---- */

/* Largest boxcar width dedisp_matched_filter accepts. */
#define DEDISP_MF_MAX_WIDTH 8192

/* Baseline removal by running mean, then boxcar matched filters, over nrows
 * independent time series of nsamps samples (Sec. 2.3 "compute a running
 * mean for the data with a given window size ... and then subtracting this off the
 * original data ... exploit a parallel prefix sum ... subtracting the points at plus
 * and minus the window radius"; "convolving the time series with boxcar
 * functions of increasing sizes (e.g., 2, 4, 8 etc. samples) ... in the same manner
 * using the parallel prefix sum").  With N = 2*radius+1 and a(t) = clip(t-radius, 0,
 * nsamps-N) (the window keeps its length and stops at the ends of the series):
 *     y[t]   = x[t] - (1/N) * sum_{k=a(t)}^{a(t)+N-1} x[k]
 *     z_w[t] = (1/sqrt(w)) * sum_{k=0}^{w-1} y[t+k]   for 0 <= t <= nsamps-w, else 0
 * (the 1/sqrt(w) keeps the white-noise variance equal for all widths).
 *   x_dev   DEVICE, [nrows][nsamps] tight, uint32 or float32 holding exact integers
 *           <= x_max (the output of dedisp_execute[_batch], any number of beams, is
 *           such an array with nrows = nbeams*ndm); 4-byte aligned.
 *   x_max   caller's upper bound on x (0 = 2^24-1; values >= 2^24 are rejected with
 *           DEDISP_ERR_OVERFLOW).  It selects 32- or 64-bit exact integer arithmetic.
 *   widths_host  HOST array of nwidths boxcar widths, 1 <= w <= min(nsamps,
 *           DEDISP_MF_MAX_WIDTH), 1 <= nwidths <= 16; copied during the call.
 *   z_dev   DEVICE float32 [nwidths][nrows][nsamps] tight, written completely.
 * All sums are exact integers; each output is fl32(numerator) * fl32(1/(N sqrt(w))),
 * i.e. within 1.5 ulp (float32) of the real value.  Only enqueues work on
 * cuda_stream.  Errors: INVALID_ARG (null or misaligned pointer, nrows/nsamps < 1,
 * nsamps > 2^30, nrows*ceil(nsamps/16384) > 2^31-1, radius < 0,
 * 2*radius+1 > nsamps, bad width or count), UNSUPPORTED_DTYPE, OVERFLOW, CUDA. */
dedisp_status dedisp_matched_filter(const void *x_dev, dedisp_out_dtype x_dtype, long long nrows,
                                    long long nsamps, int radius, const int *widths_host,
                                    int nwidths, unsigned int x_max, float *z_dev,
                                    void *cuda_stream);

/* dedisp_matched_filter that also returns the noise level of every filtered series, so that the
 * sigma-cut of dedisp_find_events needs no extra pass over z (reading R28):
 *     rms_dev[iw*nrows + r] = float32( sqrt( (1/nsamps) * sum_t z_w[r][t]^2 ) )
 * -- what dedisp_series_rms returns for the same series, up to summation order: z^2 is summed in float32
 * over the <= 64 outputs a thread writes per (width, 16 384-sample segment), then in float64 in a fixed
 * order (deterministic); relative difference to the float64 definition < 2^-20.
 *   rms_dev        DEVICE float32 [nwidths*nrows], 4-byte aligned, written completely.
 *   blockmax_dev   optional (may be NULL) DEVICE int32 [nwidths*nrows][nblocks], 4-byte aligned: a hint for
 *                  dedisp_find_events_hinted.  With (nblocks, hint_block, hint_offset) from
 *                  dedisp_matched_filter_hint_blocks(), entry [s][b] is >= the order-preserving integer
 *                  image (bits(x) for x >= 0, bits(x) ^ 0x7fffffff below) of every z[s][t] with
 *                  b*hint_block - hint_offset <= t < (b+1)*hint_block - hint_offset: the largest output of
 *                  one 2048-sample step of the kernel, gathered with warp maxima and atomicMax.
 *   workspace_dev  DEVICE scratch, 8-byte aligned, >= dedisp_matched_filter_rms_workspace_bytes();
 *                  owned by the caller, free to reuse once the call's work has completed.
 *   z_dev          may be NULL here: rms_dev (and blockmax_dev) are computed and z is not written at all
 *                  (what dedisp_search_events does in its first pass).
 * Other arguments, layouts and errors as dedisp_matched_filter; a null rms_dev, a null, misaligned
 * or too small workspace: INVALID_ARG.  Only enqueues work on cuda_stream (2 kernels, 1 memset). */
size_t dedisp_matched_filter_rms_workspace_bytes(long long nrows, long long nsamps, int nwidths);
dedisp_status dedisp_matched_filter_rms(const void *x_dev, dedisp_out_dtype x_dtype, long long nrows,
                                        long long nsamps, int radius, const int *widths_host,
                                        int nwidths, unsigned int x_max, float *z_dev, float *rms_dev,
                                        int *blockmax_dev, void *workspace_dev, size_t workspace_bytes,
                                        void *cuda_stream);
/* Blocks per series of blockmax_dev for these widths (0 on a bad argument); *hint_block and
 * *hint_offset (either may be NULL) receive the block length (2048) and the offset (largest width). */
long long dedisp_matched_filter_hint_blocks(long long nsamps, const int *widths_host, int nwidths,
                                            int *hint_block, int *hint_offset);

/* ---- peak finding ---- */

/* One detected event: a maximal run of consecutive samples of one series above threshold. */
typedef struct {
    int series;   /* row of z the run lies in */
    int t_start;  /* first sample of the run */
    int length;   /* samples in the run */
    int t_peak;   /* FIRST position of the maximum of z over the run */
    float peak;   /* that maximum */
} dedisp_event;

/* Bytes of device scratch dedisp_find_events needs for this shape (0 = shape rejected):
 * a bit mask of the sigma-cut (1 bit per sample) plus per-chunk and per-series counters. */
size_t dedisp_find_events_workspace_bytes(long long nseries, long long nsamps);

/* Sigma-cut, then contiguous regions gathered into events (Sec. 2.3 "first
 * performing a sigma-cut and then gathering contiguous regions together into individual
 * events ... 'transform' and 'reduce_by_key'"):
 *     above[s][t] = z[s][t] > nsigma * sigma[s]      (float32 product, strict >; NaN is never above)
 *     event       = maximal run of consecutive t with above[s][t], series by series
 *   z_dev      DEVICE float32 [nseries][nsamps] tight (e.g. the output of dedisp_matched_filter
 *              viewed as nwidths*nrows series); 4-byte aligned.
 *   sigma_dev  DEVICE float32 [nseries]: noise level of each series (dedisp_series_rms offers
 *              an estimate; the paper names none).
 *   workspace_dev  DEVICE scratch, 8-byte aligned, >= dedisp_find_events_workspace_bytes();
 *              owned by the caller, free to reuse after the call's work has completed.
 *   events_dev DEVICE array of max_events records (may be NULL when max_events = 0), written
 *              in ascending (series, t_start) order; events beyond max_events are dropped.
 *   count_dev  DEVICE long long, 8-byte aligned: total number of events found (may exceed
 *              max_events).
 * Only enqueues work on cuda_stream (4 kernels; z is read once, plus the samples inside runs).
 * Errors: INVALID_ARG (null/misaligned pointer, nseries/nsamps < 1, nsamps > 2^30,
 * nseries > 2^31-1, workspace too small, max_events < 0), CUDA. */
dedisp_status dedisp_find_events(const float *z_dev, long long nseries, long long nsamps,
                                 const float *sigma_dev, float nsigma, void *workspace_dev,
                                 size_t workspace_bytes, dedisp_event *events_dev,
                                 long long max_events, long long *count_dev, void *cuda_stream);

/* dedisp_find_events with a hint that lets the sigma-cut skip what cannot hold an event: hint_dev is
 * DEVICE int32 [nseries][ceil((nsamps + hint_offset) / hint_block)] with the meaning given at
 * dedisp_matched_filter_rms (blockmax_dev).  A 1024-sample chunk of z whose blocks are all at or below
 * the threshold is not read; the event list is identical to dedisp_find_events' for any valid hint
 * (entries may be larger than the true maxima, never smaller).  At a 6 sigma cut on noise nearly all of
 * z stays unread.  Errors as dedisp_find_events, plus INVALID_ARG for a null or misaligned hint,
 * hint_block < 1, hint_offset < 0. */
dedisp_status dedisp_find_events_hinted(const float *z_dev, long long nseries, long long nsamps,
                                        const float *sigma_dev, float nsigma, const int *hint_dev,
                                        int hint_block, int hint_offset, void *workspace_dev,
                                        size_t workspace_bytes, dedisp_event *events_dev,
                                        long long max_events, long long *count_dev, void *cuda_stream);

/* Rows f1 + f2 chained WITHOUT materialising z ("fusing the S/N search would remove that
 * write"; Sec. 2.3): baseline removal + boxcar filters + RMS + sigma-cut + event grouping from the
 * dedispersed series x straight to the event list.  Same definitions as dedisp_matched_filter_rms followed by
 * dedisp_find_events_hinted at threshold nsigma * rms, and the same result: the event list is identical, field by
 * field.  How: pass 1 runs the filter kernel for the RMS of every filtered series and the maxima of z over blocks of
 * 2048 outputs and stores no z; the blocks whose maximum exceeds the series' threshold (a handful at 6 sigma on
 * noise) are then re-computed by the same kernel into a compact z of max_blocks blocks (exact integer numerators, so
 * every value is bit-identical to what the dense pass writes); the sigma-cut and the grouping run on that.
 *   x_dev .. x_max   as for dedisp_matched_filter;  series index = width index * nrows + row
 *   rms_dev          float32 [nwidths * nrows] out: sqrt(mean z^2) of every filtered series
 *   max_blocks       capacity of the compact z (blocks of 2048 outputs, 8 KiB each)
 *   workspace_dev    dedisp_search_events_workspace_bytes(...) bytes, 256-byte aligned, caller-owned
 *   events_dev, max_events   as for dedisp_find_events
 *   count_dev        int64 [2] out: [0] = events found (all of them, also beyond max_events), [1] = blocks that
 *                    exceeded the threshold; the event list is complete iff count[1] <= max_blocks (else call again
 *                    with a larger max_blocks: events of the blocks that did not fit are missing)
 * Algorithmic bytes: x read once (+ 130 KB per flagged block); nothing of the size of z is written or read.
 * Only enqueues work on cuda_stream.  Errors: INVALID_ARG, UNSUPPORTED_DTYPE, OVERFLOW, CUDA. */
size_t dedisp_search_events_workspace_bytes(long long nrows, long long nsamps, const int *widths_host, int nwidths,
                                            long long max_blocks);
dedisp_status dedisp_search_events(const void *x_dev, dedisp_out_dtype x_dtype, long long nrows, long long nsamps,
                                   int radius, const int *widths_host, int nwidths, unsigned int x_max, float nsigma,
                                   float *rms_dev, long long max_blocks, void *workspace_dev, size_t workspace_bytes,
                                   dedisp_event *events_dev, long long max_events, long long *count_dev,
                                   void *cuda_stream);

/* rms_dev[s] = float32( sqrt( (1/nsamps) * sum_t z[s][t]^2 ) ), accumulated in float64: the
 * noise estimate of a baseline-removed (zero-mean) series, offered as sigma for the
 * sigma-cut (the paper does not say how sigma is obtained).  DEVICE pointers, 4-byte aligned. */
dedisp_status dedisp_series_rms(const float *z_dev, long long nseries, long long nsamps,
                                float *rms_dev, void *cuda_stream);

/* ---- multibeam coincidence RFI mask ---- */

/* PAPER.md:38-40 Sec. 2.1: "a signal exceeding 3 sigma in 4 or more beams ... a transform of the
 * multibeam time series, where for each sample the 13 beams are checked against the thresholds
 * and the result is written as a boolean RFI mask":
 *     above[b][s][t] = x[b][s][t] > fl32( mean[b][s] + fl32( nsigma * sigma[b][s] ) )
 *     mask[s][t]     = ( number of beams b with above[b][s][t] ) >= min_beams      (1 or 0)
 *   x_dev     DEVICE, nbeams blocks of [nseries][nsamps] (tight inside a beam), beam b at
 *             x_dev + b*beam_stride_bytes (a multiple of 4, >= nseries*nsamps*4); uint32 or float32
 *             holding values < 2^24 (uint32) -- e.g. the DM-0 trial of every beam of a batched
 *             dedisp_execute_batch output: nseries = 1, beam_stride_bytes = ndm*nsamps*4.
 *   mean_dev, sigma_dev  DEVICE float32 [nbeams][nseries]: level and noise of every series (the
 *             paper leaves their estimate open).
 *   mask_dev  DEVICE uint8 [nseries][nsamps], written completely.
 * Strict >, thresholds formed in float32, NaN never above.  nseries <= 65535.  Only enqueues
 * work on cuda_stream.  Errors: INVALID_ARG, UNSUPPORTED_DTYPE, CUDA. */
dedisp_status dedisp_rfi_mask(const void *x_dev, dedisp_out_dtype x_dtype, int nbeams,
                              long long nseries, long long nsamps, size_t beam_stride_bytes,
                              const float *mean_dev, const float *sigma_dev, float nsigma,
                              int min_beams, unsigned char *mask_dev, void *cuda_stream);

/* The same test when the beams live on several GPUs (the paper's deployment is one beam per GPU, and
 * the coincidence test needs all 13): every rank counts its own beams,
 *     counts[s][t] = number of LOCAL beams b with above[b][s][t]            (uint8, nbeams <= 255)
 * the counts are summed across ranks -- the path's one real exchange step: an all-reduce(SUM) of nseries*nsamps
 * bytes, done by the caller with NCCL (paper_1112_0065_b200.replicas.allreduce_beam_counts; the total number of
 * beams must stay <= 255) -- and thresholded:
 *     mask[s][t] = counts[s][t] >= min_beams.
 * dedisp_rfi_beam_counts followed by dedisp_rfi_mask_from_counts on one GPU equals dedisp_rfi_mask.
 * counts_dev / mask_dev: DEVICE uint8 [nseries][nsamps].  Errors as dedisp_rfi_mask. */
dedisp_status dedisp_rfi_beam_counts(const void *x_dev, dedisp_out_dtype x_dtype, int nbeams,
                                     long long nseries, long long nsamps, size_t beam_stride_bytes,
                                     const float *mean_dev, const float *sigma_dev, float nsigma,
                                     unsigned char *counts_dev, void *cuda_stream);
dedisp_status dedisp_rfi_mask_from_counts(const unsigned char *counts_dev, long long nseries, long long nsamps,
                                          int min_beams, unsigned char *mask_dev, void *cuda_stream);

/* A consumer of the mask (reading R39; the paper says only that the mask is "written"):
 * events whose PEAK sample is flagged are vetoed.  mask_dev is ONE series of the mask, uint8 [nsamps] (e.g. the
 * coincidence mask of the DM-0 series of all beams); an event i < min(*count_dev, max_events) with
 * mask[t_peak] != 0 gets series = -1 - series (in place, order kept, so the original index is recoverable);
 * *kept_dev (int64) = number of events left.  Events vetoed by an earlier call stay vetoed and are not counted.
 * Only enqueues work on cuda_stream.  Errors: INVALID_ARG, CUDA. */
dedisp_status dedisp_veto_events(dedisp_event *events_dev, const long long *count_dev, long long max_events,
                                 const unsigned char *mask_dev, long long nsamps, long long *kept_dev,
                                 void *cuda_stream);

/* ---- input-format variant: telescope-order stream ---- */

/* Re-lay a time-major filterbank stream (for every time sample all channels next to
 * each other, channel fastest: sample (t, c) = bits [(t*nchans + c)*nbits, +nbits) of the stream,
 * LSB-first) as the channel-major tight rows dedisp_execute reads (layouts above):
 *   in_dev   DEVICE, nsamps*nchans*nbits/8 bytes, 4-byte aligned; nchans*nbits must be a
 *            multiple of 32 (whole 32-bit words per time sample).
 *   out_dev  DEVICE, nchans rows of ceil(nsamps*nbits/8) bytes, written completely (unused high
 *            bits of a row's last byte are zero).  Pass nsamps = nsamps_out + max_delay and the
 *            result is a valid dedisp_execute input.
 * Only enqueues work on cuda_stream.  Errors: INVALID_ARG, UNSUPPORTED_NBITS, CUDA. */
dedisp_status dedisp_transpose_time_major(const void *in_dev, int nchans, long long nsamps, int nbits,
                                          void *out_dev, void *cuda_stream);

/* Diagnostics (the hazard evidence of profiles/r2_sanitizer.md; compute-sanitizer is not available on the GPU pool).
 * dedisp_debug_set_poison: byte_value 0..255 makes every later execute of the plan first fill its scratch (bit planes,
 * pair rows) with that byte, so a kernel that reads scratch words no pre-pass wrote changes its result with the
 * byte; -1 (default) switches it off.
 * dedisp_debug_checks_compiled: 1 when the library was built with -DDEDISP_CHECKS (in-kernel range and pipeline
 * checks: shared-memory read ranges, the (work item, chunk) a ring stage holds when a consumer reads it, TMA source
 * ranges, output row ranges), else 0.
 * dedisp_debug_check_errors: copies the 8 failure counters of such a build to counts_out ([0] = total, [1] =
 * shared-memory range, [2] = ring stage tag, [3] = TMA source, [4] = output range, [5] = pre-pass range); all zero
 * in a normal build.  Synchronises the device.
 * dedisp_debug_inject_fault: kind 1 makes the producer warp of a -DDEDISP_CHECKS build stamp a wrong tag on the
 * first ring stage every CTA fills (the data is still right), so that the stage-tag check must count failures --
 * the test that the checks can fail at all; kind 0 switches it off; no effect in a normal build.
 * dedisp_debug_quad_tables: HOST only, needs no GPU -- the tables dedisp_set_dm_list prepares for the quad-row path
 * (DEDISP_KERNEL_QUADS), built by the same host code from a delay table and a lane order the CALLER passes in host
 * memory, so that their addressing contract can be checked without a device (tests/test_quad_tables_cpu.py):
 *   delay_host [nchans][ndm] int32, delays in samples, >= 0, non-decreasing along the channels of a quad;
 *   lanes_host [ngroups][32] int32: the trial (column of delay_host) each lane of a DM group serves, -1 = padding lane
 *              (it repeats the last trial before it; lane 0 of a group is never padding);
 *   info       filled always: nv = variant slots per (group, quad), vslot_bytes = bytes of one variant slot of a stage,
 *              plane_words = words of one plane line of a staged box, tile_words = words per tile, nquads_pad,
 *              nrows = rows to build, usable = 0 when the list cannot take quad rows (more than nv distinct triples in
 *              a group, differences outside 0 .. 2^20 - 1, windows wider than a box) -- then nothing else is written;
 *   row0 [nquads_pad + 1], trip [nrows][4] = (d1, d2, d3, 0) of each row, vlist [ngroups][nquads_pad][nv][2] = (row or
 *   -1, first word of the variant's box for tile 0), rel [ngroups][nquads_pad][32] = (byte offset of the lane's first
 *   word in the slot << 16) | (delay & 31): each written when non-NULL (call once with NULL buffers to size them).
 * Errors: INVALID_ARG (NULL delay / lanes / info, nchans < 4, ndm < 1, ngroups < 1, a lane index outside the table,
 * tables beyond 2^28 entries). */
typedef struct {
    int nv, vslot_bytes, plane_words, tile_words, nquads_pad, nrows, usable;
} dedisp_quad_table_info;
dedisp_status dedisp_debug_quad_tables(int nchans, int ndm, const int *delay_host, int ngroups, const int *lanes_host,
                                       dedisp_quad_table_info *info, int *row0, int *trip, int *vlist,
                                       unsigned int *rel);
int dedisp_debug_checks_compiled(void);
dedisp_status dedisp_debug_inject_fault(dedisp_plan plan, int kind);
dedisp_status dedisp_debug_set_poison(dedisp_plan plan, int byte_value);
dedisp_status dedisp_debug_check_errors(dedisp_plan plan, unsigned long long *counts_out);

/* Number of kernel launches this library has issued in this process (all plans). */
unsigned long long dedisp_get_launch_count(void);

/* Last cudaError_t seen by this plan (0 = cudaSuccess) and its text. */
int dedisp_get_last_cuda_error(dedisp_plan plan);
const char *dedisp_get_error_string(dedisp_status status);

#ifdef __cplusplus
}
#endif
#endif /* DEDISP_B200_H */
