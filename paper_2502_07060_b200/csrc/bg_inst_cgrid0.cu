// bg_inst_cgrid0.cu -- complex128 instances of bg_unit_kernel (two lanes per point, 16-point tiles) for
// n = 4..10 at d = 4, 6, 8, part 1 of 2, so that these shapes do not fall to the general kernel.
#include "bg_inst_common.cuh"

BG_DEFINE_TABLE(cgrid0,
    unit_entry<C128, MM, 4, 4, 2, 2>(),
    unit_entry<C128, MM, 7, 4, 4, 2>(),
    unit_entry<C128, MM, 9, 4, 8, 2>(),
    unit_entry<C128, MM, 4, 6, 2, 2>(),
    unit_entry<C128, MM, 6, 6, 4, 2>(),
    unit_entry<C128, MM, 8, 6, 4, 2>(),
    unit_entry<C128, MM, 10, 6, 6, 2>(),      // 6 warps: two 115 KB tiles per SM (8 warps: 117 KB, one tile; 0.36 -> 0.51 of the DFMA peak)
    unit_entry<C128, MM, 5, 8, 2, 2>(),
    unit_entry<C128, MM, 7, 8, 4, 2>(),
    unit_entry<C128, MM, 9, 8, 8, 2>(),
)
