// placeholder until the tiled kernel lands: every plan falls back to DIRECT
#include "dedisp_internal.h"
dedisp_status bitslice_prepare(dedisp_plan) { return DEDISP_OK; }
void bitslice_release(dedisp_plan) {}
dedisp_status bitslice_execute(dedisp_plan, int, long long, const uint8_t *, size_t, size_t, int,
                               void *, size_t, int, cudaStream_t)
{
    return DEDISP_ERR_INVALID_ARG;
}
