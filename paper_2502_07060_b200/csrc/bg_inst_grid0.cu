// bg_inst_grid0.cu -- F_p instances of bg_unit_kernel filling the grid n = 4..10 x d = 4..10 (the dimensions
// the paper validates), part 1 of 3; split over files for build parallelism and
// the 64 KB of constant memory per module.
#include "bg_inst_common.cuh"

BG_DEFINE_TABLE(grid0,
    unit_entry<Fp31, MM, 4, 5, 1>(),
    unit_entry<Fp31, MM, 7, 5, 4>(),
    unit_entry<Fp31, MM, 10, 5, 8>(),
    unit_entry<Fp31, MM, 7, 6, 4>(),
    unit_entry<Fp31, MM, 5, 7, 1>(),
    unit_entry<Fp31, MM, 8, 7, 4>(),
    unit_entry<Fp31, MM, 4, 9, 1>(),
    unit_entry<Fp31, MM, 7, 9, 4>(),
    unit_entry<Fp31, MM, 10, 9, 8>(),
    unit_entry<Fp31, MM, 7, 10, 4>(),
)
