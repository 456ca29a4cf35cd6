// bg_inst_mont.cu -- the F_p BASELINE.json shapes over a generic 31-bit prime in Montgomery form
// (bg_field.cuh: FpMont), both metrics; every other shape runs bg_general_kernel.
#include "bg_inst_common.cuh"

BG_DEFINE_TABLE(mont,
    unit_entry<FpMont, MM, 8, 6, 4>(),
    unit_entry<FpMont, MM, 4, 4, 1>(),
    unit_entry<FpMont, MM, 10, 8, 8>(),
    unit_entry<FpMont, MM, 12, 6, 8>(),
    unit_entry<FpMont, ALT, 8, 6, 4>(),
    unit_entry<FpMont, ALT, 4, 4, 1>(),
    unit_entry<FpMont, ALT, 10, 8, 8>(),
    unit_entry<FpMont, ALT, 12, 6, 8>(),
)
