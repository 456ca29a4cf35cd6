// bg_inst_rt_fp31_mm.cu -- the run-time-n tiled kernel over Fp31, mostly-minus metric, d = 4..16; and the dispatch
#include "bg_inst_rt.cuh"

const void* bg_rt_kernel_ptr_fp31_alt(int d, int s, int w, bool multi);

const void* bg_rt_kernel_ptr_fp31(int metric, int d, int s, int w, bool multi)
{
    return metric == BG_METRIC_MOSTLY_MINUS ? rt_for_d<bg::Fp31, BG_METRIC_MOSTLY_MINUS>(d, s, w, multi)
         : metric == BG_METRIC_ALTERNATING ? bg_rt_kernel_ptr_fp31_alt(d, s, w, multi) : nullptr;
}
