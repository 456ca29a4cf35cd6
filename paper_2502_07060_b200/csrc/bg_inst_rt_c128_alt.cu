// bg_inst_rt_c128_alt.cu -- the run-time-n tiled kernel over C128, alternating metric, d = 4..16
#include "bg_inst_rt.cuh"

const void* bg_rt_kernel_ptr_c128_alt(int d, int s, int w, bool multi) { return rt_for_d<bg::C128, BG_METRIC_ALTERNATING>(d, s, w, multi); }
