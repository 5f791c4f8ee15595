// bitslice_inst_pairs8.cu -- the tiled gather-sum kernel (bitslice_kernel.cuh) on pair rows of 8-bit samples
// (geometry Cfg9P).
#include "bitslice_kernel.cuh"

dedisp_status bitslice_run_pairs8(const BitsliceCall &c)
{
    const PairTables &T = c.plan->pairs8;
    return bsk::execute_pairs<Cfg9P, 8>(c.plan, T, c.nbeams, c.nsamps_out, c.in, c.row_stride, c.in_beam_stride, c.out,
                                          c.out_beam_stride, c.out_f32, c.s, c.range, c.reserve_only);
}
