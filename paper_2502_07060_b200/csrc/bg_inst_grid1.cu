// bg_inst_grid1.cu -- F_p instances of bg_unit_kernel filling the grid n = 4..10 x d = 4..10 (the dimensions
// the paper validates), part 2 of 3; split over files for build parallelism and
// the 64 KB of constant memory per module.
#include "bg_inst_common.cuh"

BG_DEFINE_TABLE(grid1,
    unit_entry<Fp31, MM, 5, 5, 1>(),
    unit_entry<Fp31, MM, 8, 5, 4>(),
    unit_entry<Fp31, MM, 4, 6, 1>(),
    unit_entry<Fp31, MM, 10, 6, 8>(),
    unit_entry<Fp31, MM, 6, 7, 2>(),
    unit_entry<Fp31, MM, 9, 7, 4>(),
    unit_entry<Fp31, MM, 5, 9, 1>(),
    unit_entry<Fp31, MM, 8, 9, 4>(),
    unit_entry<Fp31, MM, 4, 10, 1>(),
    unit_entry<Fp31, MM, 8, 10, 4>(),
)
