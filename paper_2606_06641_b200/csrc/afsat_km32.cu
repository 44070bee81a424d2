// afsat_km32.cu -- the fp32 instantiation of the scalar register kernel k_eval_km for 9 <= k <= AFSAT_B_KMAX32
// (DESIGN.md 6.2), in a translation unit of its own so that it compiles in parallel with the
// rest (build.py).  Only built with -DAFSAT_M32_PACKED=0: by default those lengths run the packed lane-split kernel.
#define AFSAT_KM32_TU
#include "afsat_kernels.cuh"

#if !AFSAT_M32_PACKED   // with the packed lane-split kernel (the default) fp32 never launches k_eval_km beyond k = 8
namespace afsat {
template __global__ void k_eval_km<float, 9, AFSAT_B_KMAX32, 1, true, AFSAT_B_MINB>(const EvalParams<float>);
template __global__ void k_eval_km<float, 9, AFSAT_B_KMAX32, 1, false, AFSAT_B_MINB>(const EvalParams<float>);
}  // namespace afsat
#endif
