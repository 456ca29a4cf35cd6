// bg_inst_default.cu -- the kernel instances a call launches by default for the BASELINE.json shapes
// (chosen by measurement on B200)
#include "bg_inst_common.cuh"

BG_DEFINE_TABLE(default,
    unit_entry<Fp31, MM, 8, 6, 4>(),          // cfg2
    unit_entry<Fp31, MM, 4, 4, 1>(),          // cfg0
    unit_entry<Fp31, MM, 10, 8, 8>(),         // cfg3
    unit_entry<Fp31, MM, 12, 6, 8>(),         // cfg4a
    reg_entry<C128, MM, 6, 4>(),              // cfg1
    unit_entry<C128, MM, 12, 6, 12, 2>(),     // cfg4b (W = 8 / 12 / 14 / 16: 0.884 / 0.828 / 0.843 / 0.842 ms)
)
