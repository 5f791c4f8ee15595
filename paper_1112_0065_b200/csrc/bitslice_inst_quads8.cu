// bitslice_inst_quads8.cu -- the tiled gather-sum kernel (bitslice_kernel.cuh) on quad rows of 8-bit samples
// (geometry Cfg10Q).
#include "bitslice_kernel.cuh"

dedisp_status bitslice_run_quads8(const BitsliceCall &c)
{
    const QuadTables &T = c.plan->quads8;
    return bsk::execute_quads<Cfg10Q, 8>(c.plan, T, c.nbeams, c.nsamps_out, c.in, c.row_stride, c.in_beam_stride, c.out,
                                         c.out_beam_stride, c.out_f32, c.s, c.range, c.reserve_only);
}
