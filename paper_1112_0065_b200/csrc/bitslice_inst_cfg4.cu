// bitslice_inst_cfg4.cu -- the tiled gather-sum kernel (bitslice_kernel.cuh) instantiated for geometry Cfg4.
#include "bitslice_kernel.cuh"

dedisp_status bitslice_run_cfg4(const BitsliceCall &c)
{
    return bsk::execute_cfg<Cfg4>(c.plan, *c.G, c.nbeams, c.nsamps_out, c.in, c.row_stride, c.in_beam_stride, c.in_nbits,
                                 c.tscrunch, c.out, c.out_beam_stride, c.out_f32, c.s, c.range, c.reserve_only);
}
