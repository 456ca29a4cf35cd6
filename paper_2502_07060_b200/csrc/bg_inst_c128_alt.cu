// bg_inst_c128_alt.cu -- alternative complex128 instances for A/B runs (bg_set_kernel_override)
#include "bg_inst_common.cuh"

BG_DEFINE_TABLE(c128_alt,
    unit_entry<C128, MM, 6, 4, 2, 2>(),       // also the cfg1 shape with several state configurations
    unit_entry<C128, MM, 6, 4, 4, 2>(),
    unit_entry<C128, MM, 6, 4, 2, 1>(),
    unit_entry<C128, MM, 6, 4, 4, 1>(),
    unit_entry<C128, MM, 12, 6, 8, 2>(),
    unit_entry<C128, MM, 12, 6, 4, 2>(),
    unit_entry<C128, MM, 12, 6, 16, 2>(),
)
