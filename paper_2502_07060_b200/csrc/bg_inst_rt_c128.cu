// bg_inst_rt_c128.cu -- the run-time-n tiled kernel over C128, both metrics, d = 4..16
#include "bg_inst_rt.cuh"

const void* bg_rt_kernel_ptr_c128(int metric, int d, int s) { return rt_for<bg::C128>(metric, d, s); }
