// bg_inst_rt_mont.cu -- the run-time-n tiled kernel over FpMont, both metrics, d = 4..16
#include "bg_inst_rt.cuh"

const void* bg_rt_kernel_ptr_mont(int metric, int d, int s) { return rt_for<bg::FpMont>(metric, d, s); }
