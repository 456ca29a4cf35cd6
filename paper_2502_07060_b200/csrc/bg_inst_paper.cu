// bg_inst_paper.cu -- F_p instances of the fast path for the shapes of the paper's own benchmarks
// (Figs. 1-4: n = 6, 8, 9 legs in d = 4, and the dimension scans of n = 6 and
// n = 9 up to d = 10, d = 8 for the leg scan), so that they do not fall to the general kernel.
#include "bg_inst_common.cuh"

const SweepEntry* bg_entries_paper(int* count)
{
    static const SweepEntry table[] = {
        unit_entry<Fp31, 6, 4, 2>(BG_FIELD_FP31),
        unit_entry<Fp31, 8, 4, 4>(BG_FIELD_FP31),
        unit_entry<Fp31, 9, 4, 4>(BG_FIELD_FP31),
        unit_entry<Fp31, 6, 6, 2>(BG_FIELD_FP31),
        unit_entry<Fp31, 9, 6, 4>(BG_FIELD_FP31),
        unit_entry<Fp31, 6, 8, 2>(BG_FIELD_FP31),
        unit_entry<Fp31, 8, 8, 4>(BG_FIELD_FP31),
        unit_entry<Fp31, 9, 8, 4>(BG_FIELD_FP31),
        unit_entry<Fp31, 6, 10, 2>(BG_FIELD_FP31),
        unit_entry<Fp31, 9, 10, 4>(BG_FIELD_FP31),
        // the rest of the leg scans n = 4..10 at d = 4 and d = 8 (the configs cover (4,4), (10,8))
        unit_entry<Fp31, 5, 4, 1>(BG_FIELD_FP31),
        unit_entry<Fp31, 7, 4, 4>(BG_FIELD_FP31),
        unit_entry<Fp31, 10, 4, 8>(BG_FIELD_FP31),
        unit_entry<Fp31, 4, 8, 1>(BG_FIELD_FP31),
        unit_entry<Fp31, 5, 8, 1>(BG_FIELD_FP31),
        unit_entry<Fp31, 7, 8, 4>(BG_FIELD_FP31),
    };
    *count = (int)(sizeof(table) / sizeof(table[0]));
    return table;
}
