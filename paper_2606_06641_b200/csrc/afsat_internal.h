// afsat_internal.h -- shared between the host precompute (precompute.cpp, g++) and the CUDA
// translation unit (afsat.cu, nvcc).  Not part of the public ABI (include/afsat.h).
#pragma once
#include <stdint.h>
#include "../../include/afsat.h"

#define AFSAT_MAX_POINTS (AFSAT_MAX_LEN / 2 + 1)   // H = floor((k+1)/2) + 1 <= 33

// Host-side table of one signature (type, k, param): SURVEY.md §8(a) a0.
// rows[8*p .. 8*p+7] = { Re a, Im a, Re b, Im b, Re w, Im w, Re(w b), Im(w b) }, real points first.
struct AfsatSigHost {
    int32_t type, k, param;
    int32_t n_real, n_cplx;
    uint64_t satmask_lo, satmask_hi;     // bit tau set <=> satisfied with tau true literals
    double rows[AFSAT_MAX_POINTS * 8];
};

// Returns AFSAT_OK or AFSAT_E_*; never touches a device.
int afsat_sig_build(int32_t type, int32_t k, int32_t param, uint32_t flags, AfsatSigHost *out);

// The same for any symmetric constraint on k literals: bit tau of the mask set <=> satisfied with tau true literals.
int afsat_sig_build_mask(int32_t k, uint64_t satmask_lo, uint64_t satmask_hi, uint32_t flags, AfsatSigHost *out);

// Is the constraint satisfied with tau true literals?  (Table 1 / Table 2 semantics.)
bool afsat_sig_satisfied(int32_t type, int32_t k, int32_t param, int32_t tau);
