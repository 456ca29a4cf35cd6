// bg_inst_grid3.cu -- F_p instances of bg_unit_kernel for n = 11 and n = 12 at d = 4, 5, 6, 8 (cfg4a covers
// (12, 6)): the leg counts just above the paper's own scans, so that they do not fall to the general kernel
// (4-5 times slower at these sizes).
#include "bg_inst_common.cuh"

BG_DEFINE_TABLE(grid3,
    unit_entry<Fp31, MM, 11, 4, 8>(),
    unit_entry<Fp31, MM, 11, 5, 8>(),
    unit_entry<Fp31, MM, 11, 6, 8>(),
    unit_entry<Fp31, MM, 11, 8, 8>(),
    unit_entry<Fp31, MM, 12, 4, 8>(),
    unit_entry<Fp31, MM, 12, 5, 8>(),
    unit_entry<Fp31, MM, 12, 8, 8>(),
)
