// bg_inst_cgrid1.cu -- complex128 instances of bg_unit_kernel (two lanes per point, 16-point tiles) for
// n = 4..10 at d = 4, 6, 8, part 2 of 2, so that these shapes do not fall to the general kernel.
#include "bg_inst_common.cuh"

BG_DEFINE_TABLE(cgrid1,
    unit_entry<C128, MM, 5, 4, 2, 2>(),
    unit_entry<C128, MM, 8, 4, 4, 2>(),
    unit_entry<C128, MM, 10, 4, 8, 2>(),
    unit_entry<C128, MM, 5, 6, 2, 2>(),
    unit_entry<C128, MM, 7, 6, 4, 2>(),
    unit_entry<C128, MM, 9, 6, 8, 2>(),
    unit_entry<C128, MM, 4, 8, 2, 2>(),
    unit_entry<C128, MM, 6, 8, 4, 2>(),
    unit_entry<C128, MM, 8, 8, 4, 2>(),
    unit_entry<C128, MM, 10, 8, 8, 2>(),
)
