// bg_inst_rt_c128_mm.cu -- the run-time-n tiled kernel over C128, mostly-minus metric, d = 4..16; and the dispatch
#include "bg_inst_rt.cuh"

const void* bg_rt_kernel_ptr_c128_alt(int d, int s, int w, bool multi);

const void* bg_rt_kernel_ptr_c128(int metric, int d, int s, int w, bool multi)
{
    return metric == BG_METRIC_MOSTLY_MINUS ? rt_for_d<bg::C128, BG_METRIC_MOSTLY_MINUS>(d, s, w, multi)
         : metric == BG_METRIC_ALTERNATING ? bg_rt_kernel_ptr_c128_alt(d, s, w, multi) : nullptr;
}
