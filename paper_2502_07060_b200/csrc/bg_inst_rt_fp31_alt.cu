// bg_inst_rt_fp31_alt.cu -- the run-time-n tiled kernel over Fp31, alternating metric, d = 4..16
#include "bg_inst_rt.cuh"

const void* bg_rt_kernel_ptr_fp31_alt(int d, int s, int w, bool multi) { return rt_for_d<bg::Fp31, BG_METRIC_ALTERNATING>(d, s, w, multi); }
