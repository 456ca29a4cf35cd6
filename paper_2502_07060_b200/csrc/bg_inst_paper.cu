// bg_inst_paper.cu -- F_p instances of the fast path for the shapes of the paper's own benchmarks
// (Figs. 1-4: n = 6, 8, 9 legs in d = 4, and the dimension scans of n = 6 and
// n = 9 up to d = 10, d = 8 for the leg scan), so that they do not fall to the general kernel.
#include "bg_inst_common.cuh"

BG_DEFINE_TABLE(paper,
    unit_entry<Fp31, MM, 6, 4, 2>(),
    unit_entry<Fp31, MM, 8, 4, 4>(),
    unit_entry<Fp31, MM, 9, 4, 4>(),
    unit_entry<Fp31, MM, 6, 6, 2>(),
    unit_entry<Fp31, MM, 9, 6, 4>(),
    unit_entry<Fp31, MM, 6, 8, 2>(),
    unit_entry<Fp31, MM, 8, 8, 4>(),
    unit_entry<Fp31, MM, 9, 8, 4>(),
    unit_entry<Fp31, MM, 6, 10, 2>(),
    unit_entry<Fp31, MM, 9, 10, 4>(),
    unit_entry<Fp31, MM, 5, 4, 1>(),
    unit_entry<Fp31, MM, 7, 4, 4>(),
    unit_entry<Fp31, MM, 10, 4, 8>(),
    unit_entry<Fp31, MM, 4, 8, 1>(),
    unit_entry<Fp31, MM, 5, 8, 1>(),
    unit_entry<Fp31, MM, 7, 8, 4>(),
)
