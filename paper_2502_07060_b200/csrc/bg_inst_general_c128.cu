// bg_inst_general_c128.cu -- the run-time-n kernel over C128, both metrics, d = 4..16
#include "bg_inst_general.cuh"

const void* bg_general_kernel_ptr_c128(int metric, int d)
{
    return metric == BG_METRIC_MOSTLY_MINUS ? general_for_d<bg::C128, BG_METRIC_MOSTLY_MINUS>(d)
         : metric == BG_METRIC_ALTERNATING ? general_for_d<bg::C128, BG_METRIC_ALTERNATING>(d) : nullptr;
}
