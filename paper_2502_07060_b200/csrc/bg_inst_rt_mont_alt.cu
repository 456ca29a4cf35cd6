// bg_inst_rt_mont_alt.cu -- the run-time-n tiled kernel over FpMont, alternating metric, d = 4..16
#include "bg_inst_rt.cuh"

const void* bg_rt_kernel_ptr_mont_alt(int d, int s, int w, bool multi) { return rt_for_d<bg::FpMont, BG_METRIC_ALTERNATING>(d, s, w, multi); }
