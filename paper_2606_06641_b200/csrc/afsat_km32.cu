// afsat_km32.cu -- the fp32 instantiation of the scalar register kernel k_eval_km (SURVEY.md §8(a) a1-a5 for
// constraints of 9..64 literals), in a translation unit of its own: its per-length bodies are most
// of the build, and this way they compile in parallel with everything else (build.py).
#define AFSAT_KM32_TU
#include "afsat_kernels.cuh"

#if !AFSAT_M32_PACKED   // with the packed lane-split kernel (the default) fp32 never launches k_eval_km beyond k = 8
namespace afsat {
template __global__ void k_eval_km<float, 9, AFSAT_B_KMAX32, 1, true, AFSAT_B_MINB>(const EvalParams<float>);
template __global__ void k_eval_km<float, 9, AFSAT_B_KMAX32, 1, false, AFSAT_B_MINB>(const EvalParams<float>);
}  // namespace afsat
#endif
