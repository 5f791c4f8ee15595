// dedisp_api.cu -- the C ABI of libdedisp_b200.so (include/dedisp.h): plan
// management, argument validation, kernel dispatch.  No arithmetic of the method
// happens on the host: the delay table, the unpack, the gather-sum and the output
// conversion are all CUDA kernels.
#include <cmath>
#include <cstring>
#include <new>

#include "bitslice_common.cuh"
#include "dedisp_internal.h"

std::atomic<unsigned long long> g_launch_count{0};

namespace {

bool finite_pos(double x) { return std::isfinite(x) && x > 0.0; }
bool nbits_ok(int b) { return b == 1 || b == 2 || b == 4 || b == 8; }

dedisp_status check_exec_args(dedisp_plan plan, int nbeams, long long nsamps_out, const void *in,
                              int nbits, void *out, dedisp_out_dtype dt)
{
    if (!plan || !in || !out || nbeams < 1 || nsamps_out < 1) return DEDISP_ERR_INVALID_ARG;
    if (plan->ndm < 1 || !plan->d_delay) return DEDISP_ERR_NO_DM_LIST;
    if (!nbits_ok(nbits)) return DEDISP_ERR_UNSUPPORTED_NBITS;
    if (dt != DEDISP_OUT_U32 && dt != DEDISP_OUT_F32) return DEDISP_ERR_UNSUPPORTED_DTYPE;
    const long long maxv = (1ll << nbits) - 1;
    if ((long long)plan->nchans * maxv >= (1ll << 24)) return DEDISP_ERR_OVERFLOW;
    if (((uintptr_t)out & 3u) != 0) return DEDISP_ERR_INVALID_ARG;
    return DEDISP_OK;
}

void free_dm_state(dedisp_plan p)
{
    if (p->d_delay) cudaFree(p->d_delay);
    p->d_delay = nullptr;
    p->ndm = 0;
    p->max_delay = -1;
    p->dms.clear();
    quad_release(p);
    pair_release(p);
    bitslice_release(p);
}

}  // namespace

// ---- plan-owned scratch: growth and cross-stream ordering (dedisp_internal.h) ----
dedisp_status scratch_reserve_bytes(dedisp_plan plan, void **ptr, size_t *have, size_t need, cudaStream_t s)
{
    if (*have >= need) return DEDISP_OK;
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    if (s && cudaStreamIsCapturing(s, &cap) == cudaSuccess && cap != cudaStreamCaptureStatusNone) {
        // cudaFree / cudaMalloc are not allowed inside a capture (and a graph captured earlier would keep the old
        // pointer): the caller sizes the scratch with dedisp_reserve before capturing
        plan->last_cuda_error = (int)cudaErrorStreamCaptureUnsupported;
        return DEDISP_ERR_CUDA;
    }
    cudaFree(*ptr);      // synchronises the device: no kernel in flight still uses the old buffer
    *ptr = nullptr;
    *have = 0;
    const cudaError_t e = cudaMalloc(ptr, need);
    if (e != cudaSuccess) {
        cudaGetLastError();
        plan->last_cuda_error = (int)e;
        *ptr = nullptr;
        return DEDISP_ERR_ALLOC;
    }
    *have = need;
    return DEDISP_OK;
}

dedisp_status scratch_acquire(dedisp_plan plan, cudaStream_t s)
{
    if (!plan->scratch_ev_valid || plan->scratch_stream == s) return DEDISP_OK;
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    if (s) DEDISP_CUDA_TRY(plan, cudaStreamIsCapturing(s, &cap));
    // (a capturing stream cannot wait on an event recorded outside its capture: see scratch_release)
    if (cap == cudaStreamCaptureStatusNone) DEDISP_CUDA_TRY(plan, cudaStreamWaitEvent(s, plan->scratch_ev, 0));
    return DEDISP_OK;
}

dedisp_status scratch_release(dedisp_plan plan, cudaStream_t s)
{
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    if (s) DEDISP_CUDA_TRY(plan, cudaStreamIsCapturing(s, &cap));
    if (cap != cudaStreamCaptureStatusNone) {
        // an event recorded inside a capture cannot be waited on from outside it: a plan whose executes are captured
        // is ordered by the graph's own launch order (dedisp.h "Streams")
        plan->scratch_ev_valid = false;
        plan->scratch_stream = s;
        return DEDISP_OK;
    }
    if (!plan->scratch_ev) DEDISP_CUDA_TRY(plan, cudaEventCreateWithFlags(&plan->scratch_ev, cudaEventDisableTiming));
    DEDISP_CUDA_TRY(plan, cudaEventRecord(plan->scratch_ev, s));
    plan->scratch_stream = s;
    plan->scratch_ev_valid = true;
    return DEDISP_OK;
}

extern "C" {

dedisp_status dedisp_plan_create(dedisp_plan *plan, int nchans, double dt_s, double f_top_mhz,
                                 double df_mhz)
{
    if (!plan) return DEDISP_ERR_INVALID_ARG;
    *plan = nullptr;
    if (nchans < 1 || !finite_pos(dt_s) || !finite_pos(f_top_mhz) || !std::isfinite(df_mhz) ||
        !(df_mhz < 0.0))
        return DEDISP_ERR_INVALID_ARG;
    if (!(f_top_mhz + (double)(nchans - 1) * df_mhz > 0.0)) return DEDISP_ERR_INVALID_ARG;
    dedisp_plan p = new (std::nothrow) dedisp_plan_s;
    if (!p) return DEDISP_ERR_ALLOC;
    p->nchans = nchans;
    p->dt = dt_s;
    p->f_top = f_top_mhz;
    p->df = df_mhz;
    *plan = p;
    return DEDISP_OK;
}

dedisp_status dedisp_set_dm_list(dedisp_plan plan, const double *dms_host, int ndm)
{
    if (!plan || !dms_host || ndm < 1) return DEDISP_ERR_INVALID_ARG;
    for (int i = 0; i < ndm; ++i)
        if (!std::isfinite(dms_host[i]) || dms_host[i] < 0.0) return DEDISP_ERR_INVALID_ARG;
    DEDISP_CUDA_TRY(plan, cudaGetDevice(&plan->device));
    DEDISP_CUDA_TRY(plan, cudaDeviceGetAttribute(&plan->sm_count, cudaDevAttrMultiProcessorCount, plan->device));
    free_dm_state(plan);
    plan->dms.assign(dms_host, dms_host + ndm);

    double *d_dms = nullptr;
    int *d_flags = nullptr;  // [0] max_delay, [1] overflow
    const size_t tbl = (size_t)plan->nchans * (size_t)ndm * sizeof(int32_t);
    cudaError_t e = cudaMalloc(&d_dms, sizeof(double) * ndm);
    if (e == cudaSuccess) e = cudaMalloc(&d_flags, 2 * sizeof(int));
    if (e == cudaSuccess) e = cudaMalloc(&plan->d_delay, tbl);
    if (e != cudaSuccess) {
        plan->last_cuda_error = (int)e;
        cudaFree(d_dms);
        cudaFree(d_flags);
        free_dm_state(plan);
        return e == cudaErrorMemoryAllocation ? DEDISP_ERR_ALLOC : DEDISP_ERR_CUDA;
    }
    int flags[2] = {0, 0};
    e = cudaMemcpy(d_dms, dms_host, sizeof(double) * ndm, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemset(d_flags, 0, 2 * sizeof(int));
    if (e == cudaSuccess)
        e = launch_delay_table(plan->nchans, plan->dt, plan->f_top, plan->df, d_dms, ndm,
                               plan->d_delay, d_flags, d_flags + 1, 0);
    if (e == cudaSuccess) e = cudaMemcpy(flags, d_flags, sizeof(flags), cudaMemcpyDeviceToHost);
    cudaFree(d_dms);
    cudaFree(d_flags);
    if (e != cudaSuccess) {
        plan->last_cuda_error = (int)e;
        free_dm_state(plan);
        return DEDISP_ERR_CUDA;
    }
    if (flags[1]) {
        free_dm_state(plan);
        return DEDISP_ERR_OVERFLOW;
    }
    plan->ndm = ndm;
    plan->max_delay = flags[0];
#ifdef DEDISP_CHECKS
    if (!plan->d_check_errors) {
        DEDISP_CUDA_TRY(plan, cudaMalloc(&plan->d_check_errors, sizeof(unsigned long long) * DEDISP_NCHECK));
        DEDISP_CUDA_TRY(plan, cudaMemset(plan->d_check_errors, 0, sizeof(unsigned long long) * DEDISP_NCHECK));
    }
#endif
    dedisp_status st = bitslice_prepare(plan);
    if (st == DEDISP_OK) st = pair_prepare(plan);
    if (st == DEDISP_OK) st = quad_prepare(plan);
    if (st != DEDISP_OK) free_dm_state(plan);
    return st;
}

dedisp_status dedisp_execute_tscrunch(dedisp_plan plan, int tscrunch, int nbeams, long long nsamps_out,
                                      const void *in_dev, size_t in_beam_stride_bytes, int in_nbits,
                                      void *out_dev, size_t out_beam_stride_bytes,
                                      dedisp_out_dtype out_dtype, void *cuda_stream)
{
    dedisp_status st = check_exec_args(plan, nbeams, nsamps_out, in_dev, in_nbits, out_dev, out_dtype);
    if (st != DEDISP_OK) return st;
    if (nbeams > 1 && (out_beam_stride_bytes & 3u)) return DEDISP_ERR_INVALID_ARG;
    const long long maxv = (1ll << in_nbits) - 1;
    if (tscrunch < 1 || (tscrunch > 1 && tscrunch * maxv > 255)) return DEDISP_ERR_INVALID_ARG;
    if ((long long)plan->nchans * tscrunch * maxv >= (1ll << 24)) return DEDISP_ERR_OVERFLOW;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const size_t row_stride = dedisp_get_in_row_stride_bytes_tscrunch(plan, tscrunch, nsamps_out, in_nbits);
    const int f32 = (out_dtype == DEDISP_OUT_F32);
    const uint8_t *in = (const uint8_t *)in_dev;

    if (plan->want != DEDISP_KERNEL_DIRECT) {
        st = bitslice_execute(plan, nbeams, nsamps_out, in, row_stride, in_beam_stride_bytes,
                              in_nbits, tscrunch, out_dev, out_beam_stride_bytes, f32, s);
        if (st == DEDISP_OK) {
            plan->last_kernel = plan->bitslice_kind;
            return DEDISP_OK;
        }
        // INVALID_ARG from bitslice_execute means "plan does not fit this kernel"
        if (st != DEDISP_ERR_INVALID_ARG || plan->want == DEDISP_KERNEL_BITSLICE || plan->want == DEDISP_KERNEL_PAIRS ||
            plan->want == DEDISP_KERNEL_QUADS)
            return st;
    }
    int direct_nbits = in_nbits;
    size_t direct_beam_stride = in_beam_stride_bytes;
    size_t direct_row_stride = row_stride;
    bool uses_scratch = false;
    if (tscrunch > 1) {
        // block sums as one byte each in the plan's scratch, then the DIRECT kernel on 8-bit samples
        const long long n_scr = nsamps_out + plan->max_delay;
        const size_t need = (size_t)nbeams * plan->nchans * (size_t)n_scr;
        if (nbeams > 65535 || plan->nchans > 65535) return DEDISP_ERR_INVALID_ARG;
        st = scratch_reserve(plan, &plan->d_planes, &plan->planes_bytes, need, s);
        if (st == DEDISP_OK) st = scratch_acquire(plan, s);
        if (st != DEDISP_OK) return st;
        uses_scratch = true;
        DEDISP_CUDA_TRY(plan, launch_tscrunch_bytes(in_nbits, tscrunch, in, in_beam_stride_bytes, row_stride,
                                                    plan->nchans, nbeams, n_scr, (uint8_t *)plan->d_planes, s));
        in = (const uint8_t *)plan->d_planes;
        direct_nbits = 8;
        direct_row_stride = (size_t)n_scr;
        direct_beam_stride = (size_t)plan->nchans * (size_t)n_scr;
    }
    if (plan->timing) cudaEventRecord(plan->ev[2], s);
    // grid.z limit of the direct kernel
    for (int b0 = 0; b0 < nbeams; b0 += 65535) {
        const int nb = (nbeams - b0 < 65535) ? nbeams - b0 : 65535;
        DEDISP_CUDA_TRY(plan, launch_direct(plan->d_delay, plan->nchans, plan->ndm, nsamps_out,
                                            in + (size_t)b0 * direct_beam_stride, direct_row_stride,
                                            direct_beam_stride, direct_nbits,
                                            (uint8_t *)out_dev + (size_t)b0 * out_beam_stride_bytes,
                                            out_beam_stride_bytes, f32, nb, s));
    }
    if (plan->timing) {
        cudaEventRecord(plan->ev[3], s);
        plan->timing_valid = true;
        plan->timing_has_prepass = false;
    }
    plan->last_kernel = DEDISP_KERNEL_DIRECT;
    return uses_scratch ? scratch_release(plan, s) : DEDISP_OK;
}

dedisp_status dedisp_execute_batch(dedisp_plan plan, int nbeams, long long nsamps_out,
                                   const void *in_dev, size_t in_beam_stride_bytes, int in_nbits,
                                   void *out_dev, size_t out_beam_stride_bytes,
                                   dedisp_out_dtype out_dtype, void *cuda_stream)
{
    return dedisp_execute_tscrunch(plan, 1, nbeams, nsamps_out, in_dev, in_beam_stride_bytes, in_nbits, out_dev,
                                   out_beam_stride_bytes, out_dtype, cuda_stream);
}

dedisp_status dedisp_execute(dedisp_plan plan, long long nsamps_out, const void *in_dev,
                             int in_nbits, void *out_dev, dedisp_out_dtype out_dtype,
                             void *cuda_stream)
{
    return dedisp_execute_batch(plan, 1, nsamps_out, in_dev, 0, in_nbits, out_dev, 0, out_dtype,
                                cuda_stream);
}

dedisp_status dedisp_reserve(dedisp_plan plan, int nbeams, long long nsamps_out, int in_nbits)
{
    if (!plan || nbeams < 1 || nsamps_out < 1) return DEDISP_ERR_INVALID_ARG;
    if (plan->ndm < 1 || !plan->d_delay) return DEDISP_ERR_NO_DM_LIST;
    if (!nbits_ok(in_nbits)) return DEDISP_ERR_UNSUPPORTED_NBITS;
    if (plan->want == DEDISP_KERNEL_DIRECT) return DEDISP_OK;       // the DIRECT kernel has no scratch
    const size_t row_stride = dedisp_get_in_row_stride_bytes(plan, nsamps_out, in_nbits);
    const dedisp_status st = bitslice_execute(plan, nbeams, nsamps_out, (const uint8_t *)nullptr, row_stride, 0, in_nbits,
                                              1, nullptr, 0, 0, nullptr, nullptr, true);
    // INVALID_ARG: the plan does not fit the tiled kernel; AUTO then runs DIRECT, which needs nothing
    return (st == DEDISP_ERR_INVALID_ARG && plan->want == DEDISP_KERNEL_AUTO) ? DEDISP_OK : st;
}

dedisp_status dedisp_execute_host(dedisp_plan plan, int nbeams, long long nsamps_out,
                                  const void *in_host, int in_nbits, void *out_host,
                                  dedisp_out_dtype out_dtype)
{
    if (!plan || !in_host || !out_host || nbeams < 1 || nsamps_out < 1) return DEDISP_ERR_INVALID_ARG;
    if (plan->ndm < 1) return DEDISP_ERR_NO_DM_LIST;
    if (!nbits_ok(in_nbits)) return DEDISP_ERR_UNSUPPORTED_NBITS;
    const size_t row = dedisp_get_in_row_stride_bytes(plan, nsamps_out, in_nbits);
    const size_t in_beam = row * (size_t)plan->nchans;
    const size_t out_beam = (size_t)plan->ndm * (size_t)nsamps_out * 4;
    const size_t in_bytes = in_beam * nbeams, out_bytes = out_beam * nbeams;
    if (!plan->host_stream)
        DEDISP_CUDA_TRY(plan, cudaStreamCreateWithFlags(&plan->host_stream, cudaStreamNonBlocking));
    cudaStream_t s = plan->host_stream;
    dedisp_status sst = scratch_reserve(plan, &plan->d_in_stage, &plan->in_stage_bytes, in_bytes, s);
    if (sst == DEDISP_OK) sst = scratch_reserve(plan, &plan->d_out_stage, &plan->out_stage_bytes, out_bytes, s);
    if (sst != DEDISP_OK) return sst;      // (the failed cudaMalloc is cleared and recorded in last_cuda_error)
    DEDISP_CUDA_TRY(plan, cudaMemcpyAsync(plan->d_in_stage, in_host, in_bytes, cudaMemcpyHostToDevice, s));
    // The result (out_bytes) dominates the transfer time, so it leaves in pieces while the kernel is
    // still running: one beam at a time, or -- single beam, trial DMs given in ascending order, so that
    // a range of DM groups is a range of output rows -- one range of DM groups at a time.  Each piece is
    // copied on a second stream as soon as its kernel has finished.
    const int ngroups = plan->want == DEDISP_KERNEL_DIRECT ? 0 : bitslice_ngroups(plan, in_nbits);
    const bool by_beam = ngroups > 0 && nbeams > 1;
    const bool by_range = ngroups >= 2 && nbeams == 1 && plan->order_identity;
    if (by_beam || by_range) {
        dedisp_status chk = check_exec_args(plan, nbeams, nsamps_out, plan->d_in_stage, in_nbits, plan->d_out_stage,
                                            out_dtype);
        if (chk != DEDISP_OK) return chk;
        constexpr int NEV = (int)(sizeof(plan->chunk_ev) / sizeof(plan->chunk_ev[0]));
        if (!plan->copy_stream)
            DEDISP_CUDA_TRY(plan, cudaStreamCreateWithFlags(&plan->copy_stream, cudaStreamNonBlocking));
        for (int i = 0; i < NEV; ++i)
            if (!plan->chunk_ev[i])
                DEDISP_CUDA_TRY(plan, cudaEventCreateWithFlags(&plan->chunk_ev[i], cudaEventDisableTiming));
        const int f32 = (out_dtype == DEDISP_OUT_F32);
        const int nchunks = by_beam ? nbeams : (ngroups < 8 ? ngroups : 8);
        const size_t row_bytes = (size_t)nsamps_out * 4;
        for (int c = 0; c < nchunks; ++c) {
            size_t off, bytes;
            dedisp_status st;
            if (by_beam) {
                off = (size_t)c * out_beam;
                bytes = out_beam;
                st = bitslice_execute(plan, 1, nsamps_out, (const uint8_t *)plan->d_in_stage + (size_t)c * in_beam,
                                      row, 0, in_nbits, 1, (uint8_t *)plan->d_out_stage + off, 0, f32, s);
            } else {
                BitsliceRange rg;
                rg.g_begin = (int)((long long)ngroups * c / nchunks);
                rg.g_count = (int)((long long)ngroups * (c + 1) / nchunks) - rg.g_begin;
                rg.prepass = (c == 0);
                const long long d0 = 32ll * rg.g_begin;
                long long d1 = d0 + 32ll * rg.g_count;
                if (d1 > plan->ndm) d1 = plan->ndm;
                off = (size_t)d0 * row_bytes;
                bytes = (size_t)(d1 - d0) * row_bytes;
                st = bitslice_execute(plan, 1, nsamps_out, (const uint8_t *)plan->d_in_stage, row, 0, in_nbits, 1,
                                      plan->d_out_stage, 0, f32, s, &rg);
            }
            if (st != DEDISP_OK) return st;
            cudaEvent_t ev = plan->chunk_ev[c % NEV];
            if (c >= NEV) DEDISP_CUDA_TRY(plan, cudaEventSynchronize(ev));   // its earlier use has been consumed
            DEDISP_CUDA_TRY(plan, cudaEventRecord(ev, s));
            DEDISP_CUDA_TRY(plan, cudaStreamWaitEvent(plan->copy_stream, ev, 0));
            DEDISP_CUDA_TRY(plan, cudaMemcpyAsync((uint8_t *)out_host + off, (uint8_t *)plan->d_out_stage + off, bytes,
                                                  cudaMemcpyDeviceToHost, plan->copy_stream));
        }
        plan->last_kernel = plan->bitslice_kind;
        DEDISP_CUDA_TRY(plan, cudaStreamSynchronize(s));
        DEDISP_CUDA_TRY(plan, cudaStreamSynchronize(plan->copy_stream));
        return DEDISP_OK;
    }
    dedisp_status st = dedisp_execute_batch(plan, nbeams, nsamps_out, plan->d_in_stage, in_beam,
                                            in_nbits, plan->d_out_stage, out_beam, out_dtype, s);
    if (st != DEDISP_OK) return st;
    DEDISP_CUDA_TRY(plan, cudaMemcpyAsync(out_host, plan->d_out_stage, out_bytes, cudaMemcpyDeviceToHost, s));
    DEDISP_CUDA_TRY(plan, cudaStreamSynchronize(s));
    return DEDISP_OK;
}

dedisp_status dedisp_destroy(dedisp_plan plan)
{
    if (!plan) return DEDISP_OK;
    free_dm_state(plan);
    cudaFree(plan->d_pair_rows);
    cudaFree(plan->d_check_errors);
    cudaFree(plan->d_planes);
    cudaFree(plan->d_in_stage);
    cudaFree(plan->d_out_stage);
    if (plan->host_stream) cudaStreamDestroy(plan->host_stream);
    if (plan->copy_stream) cudaStreamDestroy(plan->copy_stream);
    for (cudaEvent_t e : plan->chunk_ev)
        if (e) cudaEventDestroy(e);
    for (int i = 0; i < 4; ++i)
        if (plan->ev[i]) cudaEventDestroy(plan->ev[i]);
    if (plan->scratch_ev) cudaEventDestroy(plan->scratch_ev);
    delete plan;
    return DEDISP_OK;
}

int dedisp_get_max_delay(dedisp_plan plan) { return (plan && plan->ndm > 0) ? plan->max_delay : -1; }
int dedisp_get_nchans(dedisp_plan plan) { return plan ? plan->nchans : 0; }
int dedisp_get_ndm(dedisp_plan plan) { return plan ? plan->ndm : 0; }

size_t dedisp_get_in_row_stride_bytes(dedisp_plan plan, long long nsamps_out, int in_nbits)
{
    if (!plan || plan->ndm < 1 || nsamps_out < 1 || !nbits_ok(in_nbits)) return 0;
    const unsigned long long n = (unsigned long long)nsamps_out + (unsigned long long)plan->max_delay;
    return (size_t)((n * (unsigned)in_nbits + 7) / 8);
}

size_t dedisp_get_in_row_stride_bytes_tscrunch(dedisp_plan plan, int tscrunch, long long nsamps_out, int in_nbits)
{
    if (!plan || plan->ndm < 1 || nsamps_out < 1 || tscrunch < 1 || !nbits_ok(in_nbits)) return 0;
    const unsigned long long n = (unsigned long long)nsamps_out + (unsigned long long)plan->max_delay;
    return (size_t)((n * (unsigned)tscrunch * (unsigned)in_nbits + 7) / 8);
}

dedisp_status dedisp_get_delay_table(dedisp_plan plan, int *host_out)
{
    if (!plan || !host_out) return DEDISP_ERR_INVALID_ARG;
    if (plan->ndm < 1 || !plan->d_delay) return DEDISP_ERR_NO_DM_LIST;
    DEDISP_CUDA_TRY(plan, cudaMemcpy(host_out, plan->d_delay,
                                     (size_t)plan->nchans * plan->ndm * sizeof(int32_t),
                                     cudaMemcpyDeviceToHost));
    return DEDISP_OK;
}

dedisp_status dedisp_set_kernel(dedisp_plan plan, dedisp_kernel which)
{
    if (!plan || (int)which < 0 || (int)which > 4) return DEDISP_ERR_INVALID_ARG;
    plan->want = which;
    return DEDISP_OK;
}

dedisp_status dedisp_set_timing(dedisp_plan plan, int enable)
{
    if (!plan) return DEDISP_ERR_INVALID_ARG;
    if (enable)
        for (int i = 0; i < 4; ++i)
            if (!plan->ev[i]) DEDISP_CUDA_TRY(plan, cudaEventCreate(&plan->ev[i]));
    plan->timing = enable != 0;
    plan->timing_valid = false;
    return DEDISP_OK;
}

dedisp_status dedisp_get_last_kernel_ms(dedisp_plan plan, float *prepass_ms, float *main_ms)
{
    if (!plan || !prepass_ms || !main_ms) return DEDISP_ERR_INVALID_ARG;
    if (!plan->timing || !plan->timing_valid) return DEDISP_ERR_INVALID_ARG;
    *prepass_ms = 0.f;
    DEDISP_CUDA_TRY(plan, cudaEventSynchronize(plan->ev[3]));
    DEDISP_CUDA_TRY(plan, cudaEventElapsedTime(main_ms, plan->ev[2], plan->ev[3]));
    if (plan->timing_has_prepass)
        DEDISP_CUDA_TRY(plan, cudaEventElapsedTime(prepass_ms, plan->ev[0], plan->ev[1]));
    return DEDISP_OK;
}

int dedisp_debug_checks_compiled(void)
{
#ifdef DEDISP_CHECKS
    return 1;
#else
    return 0;
#endif
}

dedisp_status dedisp_debug_set_poison(dedisp_plan plan, int byte_value)
{
    if (!plan || byte_value < -1 || byte_value > 255) return DEDISP_ERR_INVALID_ARG;
    plan->poison = byte_value;
    return DEDISP_OK;
}

dedisp_status dedisp_debug_inject_fault(dedisp_plan plan, int kind)
{
    if (!plan || kind < 0 || kind > 1) return DEDISP_ERR_INVALID_ARG;
    plan->inject_fault = kind;
    return DEDISP_OK;
}

dedisp_status dedisp_debug_check_errors(dedisp_plan plan, unsigned long long *counts_out)
{
    if (!plan || !counts_out) return DEDISP_ERR_INVALID_ARG;
    for (int i = 0; i < DEDISP_NCHECK; ++i) counts_out[i] = 0;
    if (plan->d_check_errors)      // (synchronises with the kernels that may still be counting)
        DEDISP_CUDA_TRY(plan, cudaMemcpy(counts_out, plan->d_check_errors, sizeof(unsigned long long) * DEDISP_NCHECK,
                                         cudaMemcpyDeviceToHost));
    return DEDISP_OK;
}

int dedisp_get_last_kernel(dedisp_plan plan) { return plan ? plan->last_kernel : 0; }
unsigned long long dedisp_get_launch_count(void) { return g_launch_count.load(); }
int dedisp_get_last_cuda_error(dedisp_plan plan) { return plan ? plan->last_cuda_error : 0; }

const char *dedisp_get_error_string(dedisp_status s)
{
    switch (s) {
        case DEDISP_OK: return "ok";
        case DEDISP_ERR_INVALID_ARG: return "invalid argument";
        case DEDISP_ERR_NO_DM_LIST: return "no DM list set";
        case DEDISP_ERR_UNSUPPORTED_NBITS: return "unsupported in_nbits (1, 2, 4 or 8)";
        case DEDISP_ERR_UNSUPPORTED_DTYPE: return "unsupported output dtype";
        case DEDISP_ERR_OVERFLOW: return "sum or delay out of range";
        case DEDISP_ERR_ALLOC: return "allocation failed";
        case DEDISP_ERR_CUDA: return "CUDA error";
        case DEDISP_ERR_SCRATCH_LIMIT: return "problem exceeds the 32 MiB static scratch of dedisp_execute_static";
    }
    return "unknown status";
}

}  // extern "C"
