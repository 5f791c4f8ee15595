// static_scratch.cu -- dedisp_execute_static: dedispersion of one beam that allocates NOTHING.
//
//   out[d][t] = sum_c in[c][t + delay[c][d]]       (BASELINE.json:north_star)
//
// Why: some callers cannot call cudaMalloc -- code under CUDA-graph capture, tight serving loops, harnesses that
// forbid it.  dedisp_execute grows the plan's bit-plane scratch with cudaFree + cudaMalloc on demand (dedisp_reserve
// moves that ahead of time, but still allocates).  This entry point runs the same plain tiled kernel
// (DEDISP_KERNEL_BITSLICE: unpack pre-pass -> bit planes -> TMA-staged gather-sum) with the bit planes in a
// FILE-SCOPE device array of fixed size, DEDISP_STATIC_SCRATCH_BYTES = 32 MiB: enough for the HTRU gulp (1024 channels
// x 2 bits x 86 012 samples = 23.3 MB of planes), far too small for the 8-bit wideband config (750 MB), which is
// rejected with DEDISP_ERR_SCRATCH_LIMIT.  Every GPU that loads the library holds the 32 MiB until the process exits
// (CUDA loads modules lazily: the driver reserves them when this translation unit's module is first touched on a
// device, i.e. at the first call there -- make that call outside a graph capture).
//
// The array is shared by every call, plan and stream of the process and keeps the last call's contents.  Nothing has
// to start at zero: the pre-pass writes every word of every (padded) channel row the kernel stages, so stale words of
// an earlier, larger call lie outside what a later call reads (tests/test_zz_no_alloc.py runs a large call, then a
// small one).  Calls that overlap on the GPU -- two streams, two plans, two host threads -- RACE on the array: the
// caller serialises them (one stream, or events).  The pair-row path is not offered here: its rows need 373 MB for the
// gulp.
//
// Host code must not hand `g_static_planes` itself to a kernel: in host code that name is a host-side stand-in, not a
// device address.  The address comes from cudaGetSymbolAddress, once per device, with that device current.
#include <mutex>

#include "bitslice_common.cuh"
#include "dedisp_internal.h"

using namespace bs;

namespace {

constexpr size_t STATIC_BYTES = (size_t)DEDISP_STATIC_SCRATCH_BYTES;
static __device__ __align__(256) uint32_t g_static_planes[STATIC_BYTES / 4];

constexpr int MAX_DEVICES = 64;
std::mutex g_addr_mutex;
void *g_addr[MAX_DEVICES] = {};      // device address of g_static_planes on each device, resolved once

// Device address of the array on the CURRENT device (set-up: the first call on a device resolves it; no allocation --
// the array is part of the module image).
cudaError_t static_planes_address(int device, void **ptr)
{
    if (device < 0 || device >= MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_addr_mutex);
    if (!g_addr[device]) {
        void *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_static_planes);
        if (e != cudaSuccess) return e;
        if (!p || ((uintptr_t)p & 255u)) return cudaErrorInvalidSymbol;
        g_addr[device] = p;
    }
    *ptr = g_addr[device];
    return cudaSuccess;
}

// bytes of bit planes execute_cfg<C> needs for one beam (the formula of bitslice_kernel.cuh::execute_cfg)
template <class C>
unsigned long long planes_need(const dedisp_plan_s *plan, const BitsliceGeom &G, long long nsamps_out)
{
    const long long ntiles = (nsamps_out + C::TILE_SAMPS - 1) / C::TILE_SAMPS;
    const long long pitch = (((long long)(plan->max_delay >> 5) + ntiles * C::TILE_WORDS + G.win_words + 4) + 3) & ~3ll;
    return (unsigned long long)G.nchans_pad * C::NB * (unsigned long long)pitch * 4ull;
}

// the plan's scratch pointer for the duration of one call (a plan is not thread-safe: dedisp.h "Threading")
struct ScratchSwap {
    dedisp_plan plan;
    uint32_t *ptr;
    size_t bytes;
    ScratchSwap(dedisp_plan p, void *stat) : plan(p), ptr(p->d_planes), bytes(p->planes_bytes)
    {
        p->d_planes = (uint32_t *)stat;
        p->planes_bytes = STATIC_BYTES;
    }
    ~ScratchSwap()
    {
        plan->d_planes = ptr;
        plan->planes_bytes = bytes;
    }
};

}  // namespace

extern "C" size_t dedisp_static_scratch_bytes(void) { return STATIC_BYTES; }

extern "C" dedisp_status dedisp_execute_static(dedisp_plan plan, long long nsamps_out, const void *in_dev, int in_nbits,
                                               void *out_dev, dedisp_out_dtype out_dtype, void *cuda_stream)
{
    if (!plan || !in_dev || !out_dev || nsamps_out < 1) return DEDISP_ERR_INVALID_ARG;
    if (plan->ndm < 1 || !plan->d_delay) return DEDISP_ERR_NO_DM_LIST;
    if (in_nbits != 1 && in_nbits != 2 && in_nbits != 4 && in_nbits != 8) return DEDISP_ERR_UNSUPPORTED_NBITS;
    if (out_dtype != DEDISP_OUT_U32 && out_dtype != DEDISP_OUT_F32) return DEDISP_ERR_UNSUPPORTED_DTYPE;
    const long long maxv = (1ll << in_nbits) - 1;
    if ((long long)plan->nchans * maxv >= (1ll << 24)) return DEDISP_ERR_OVERFLOW;
    if (((uintptr_t)out_dev & 3u) != 0) return DEDISP_ERR_INVALID_ARG;
    // the plain tiled kernel must be able to serve the plan (it can for every plan the bit-sliced tables were built
    // for); there is no DIRECT fallback here
    const BitsliceGeom &G = plan->geom[geom_index(in_nbits)];
    if (!G.usable || CH_PAD * maxv >= (1ll << G.nplanes_acc) || G.nchans_pad > 65535) return DEDISP_ERR_INVALID_ARG;
    const unsigned long long need = in_nbits == 1   ? planes_need<Cfg1>(plan, G, nsamps_out)
                                    : in_nbits == 2 ? planes_need<Cfg2>(plan, G, nsamps_out)
                                    : in_nbits == 4 ? planes_need<Cfg4>(plan, G, nsamps_out)
                                                    : planes_need<Cfg8>(plan, G, nsamps_out);
    if (need > STATIC_BYTES) return DEDISP_ERR_SCRATCH_LIMIT;
    int device = 0;
    DEDISP_CUDA_TRY(plan, cudaGetDevice(&device));
    if (device != plan->device) return DEDISP_ERR_INVALID_ARG;      // the plan's tables live on the device of set_dm_list
    void *stat = nullptr;
    DEDISP_CUDA_TRY(plan, static_planes_address(device, &stat));

    cudaStream_t s = (cudaStream_t)cuda_stream;
    const size_t row_stride = dedisp_get_in_row_stride_bytes(plan, nsamps_out, in_nbits);
    const BitsliceCall call = {plan, &G, 1, nsamps_out, (const uint8_t *)in_dev, row_stride, 0, in_nbits, 1, out_dev,
                               0, out_dtype == DEDISP_OUT_F32, s, BitsliceRange(), false};
    dedisp_status st;
    {
        ScratchSwap swap(plan, stat);      // execute_cfg finds planes_bytes >= need: it neither frees nor allocates
        st = in_nbits == 1 ? bitslice_run_cfg1(call) : in_nbits == 2 ? bitslice_run_cfg2(call)
             : in_nbits == 4 ? bitslice_run_cfg4(call) : bitslice_run_cfg8(call);
    }
    if (st == DEDISP_OK) plan->last_kernel = DEDISP_KERNEL_BITSLICE;
    return st;
}
