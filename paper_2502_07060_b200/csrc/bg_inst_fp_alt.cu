// bg_inst_fp_alt.cu -- alternative F_p instances for A/B runs (bg_set_kernel_override)
#include "bg_inst_common.cuh"

BG_DEFINE_TABLE(fp_alt,
    unit_entry<Fp31, MM, 8, 6, 6>(),
    unit_entry<Fp31, MM, 8, 6, 2>(),
    unit_entry<Fp31, MM, 10, 8, 4>(),
    unit_entry<Fp31, MM, 12, 6, 16>(),
    unit_entry<Fp31, MM, 12, 6, 4>(),
)
