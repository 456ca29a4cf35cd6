// bg_host_util.h -- host helpers shared by the translation units of libbg_b200 (defined in bg_api.cu)
#pragma once
#include <stdint.h>

#include "bg_field.cuh"

// Montgomery constants of prime p into slot i; false unless p is odd and 2^30 < p < 2^31
bool bg_mont_constants(uint32_t p, int i, bg::FpMont::Params* q);

// The two spinor constants of bg_states.cuh over F_p, in the kernels' internal form (plain residues
// when q == NULL, Montgomery form of slot 0 of q otherwise): alternating metric jm = -1, jv = 1;
// mostly-minus metric jm = jv = sqrt(-1), which exists only when p = 1 mod 4 (false otherwise:
// 2^31-1 = 3 mod 4 has none, which is why the paper switches to the alternating metric).
bool bg_spinor_consts_fp(uint32_t p, int metric, const bg::FpMont::Params* q, uint32_t* jm, uint32_t* jv);
