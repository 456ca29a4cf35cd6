// bg_inst_metric.cu -- the BASELINE.json shapes with Caravel's alternating metric diag(1,-1,1,-1,..)
// over F_p (p = 2^31-1) and complex128; every other shape runs bg_general_kernel.
#include "bg_inst_common.cuh"

BG_DEFINE_TABLE(metric,
    unit_entry<Fp31, ALT, 8, 6, 4>(),
    unit_entry<Fp31, ALT, 4, 4, 1>(),
    unit_entry<Fp31, ALT, 10, 8, 8>(),
    unit_entry<Fp31, ALT, 12, 6, 8>(),
    unit_entry<C128, ALT, 6, 4, 2, 2>(),
    unit_entry<C128, ALT, 12, 6, 8, 2>(),
)
