// bg_inst_rt_mont_mm.cu -- the run-time-n tiled kernel over FpMont, mostly-minus metric, d = 4..16; and the dispatch
#include "bg_inst_rt.cuh"

const void* bg_rt_kernel_ptr_mont_alt(int d, int s, int w, bool multi);

const void* bg_rt_kernel_ptr_mont(int metric, int d, int s, int w, bool multi)
{
    return metric == BG_METRIC_MOSTLY_MINUS ? rt_for_d<bg::FpMont, BG_METRIC_MOSTLY_MINUS>(d, s, w, multi)
         : metric == BG_METRIC_ALTERNATING ? bg_rt_kernel_ptr_mont_alt(d, s, w, multi) : nullptr;
}
