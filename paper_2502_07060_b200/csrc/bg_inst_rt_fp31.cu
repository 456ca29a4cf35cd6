// bg_inst_rt_fp31.cu -- the run-time-n tiled kernel over Fp31, both metrics, d = 4..16
#include "bg_inst_rt.cuh"

const void* bg_rt_kernel_ptr_fp31(int metric, int d, int s) { return rt_for<bg::Fp31>(metric, d, s); }
