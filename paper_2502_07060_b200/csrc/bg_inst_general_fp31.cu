// bg_inst_general_fp31.cu -- the run-time-n kernel over Fp31, both metrics, d = 4..16
#include "bg_inst_general.cuh"

const void* bg_general_kernel_ptr_fp31(int metric, int d)
{
    return metric == BG_METRIC_MOSTLY_MINUS ? general_for_d<bg::Fp31, BG_METRIC_MOSTLY_MINUS>(d)
         : metric == BG_METRIC_ALTERNATING ? general_for_d<bg::Fp31, BG_METRIC_ALTERNATING>(d) : nullptr;
}
