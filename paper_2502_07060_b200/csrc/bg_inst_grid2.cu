// bg_inst_grid2.cu -- F_p instances of bg_unit_kernel filling the grid n = 4..10 x d = 4..10 (the dimensions
// the paper validates), part 3 of 3; split over files for build parallelism and
// the 64 KB of constant memory per module.
#include "bg_inst_common.cuh"

BG_DEFINE_TABLE(grid2,
    unit_entry<Fp31, MM, 6, 5, 2>(),
    unit_entry<Fp31, MM, 9, 5, 4>(),
    unit_entry<Fp31, MM, 5, 6, 1>(),
    unit_entry<Fp31, MM, 4, 7, 1>(),
    unit_entry<Fp31, MM, 7, 7, 4>(),
    unit_entry<Fp31, MM, 10, 7, 8>(),
    unit_entry<Fp31, MM, 6, 9, 2>(),
    unit_entry<Fp31, MM, 9, 9, 4>(),
    unit_entry<Fp31, MM, 5, 10, 1>(),
    unit_entry<Fp31, MM, 10, 10, 8>(),
)
