// afsat_ks32.cu -- the instantiation of the lane-split register kernel k_eval_split (SURVEY.md §8(a) a1-a5 for fp32
// constraints longer than AFSAT_B_KMAX32 literals), in a translation unit of its own so that its
// per-length bodies compile in parallel with the rest of the build (build.py).
#define AFSAT_KM32_TU   // the non-template kernels of afsat_kernels.cuh are defined in afsat.cu only
#define AFSAT_KS32_TU
#include "afsat_split.cuh"

namespace afsat {
template __global__ void k_eval_split<float, AFSAT_L32_KMIN, AFSAT_MAX_LEN, AFSAT_L32_NS, 1, true, AFSAT_L32_THREADS, AFSAT_L32_MINB>(const EvalParams<float>);
template __global__ void k_eval_split<float, AFSAT_L32_KMIN, AFSAT_MAX_LEN, AFSAT_L32_NS, 1, false, AFSAT_L32_THREADS, AFSAT_L32_MINB>(const EvalParams<float>);
#if AFSAT_L64_SPLIT
template __global__ void k_eval_split<double, AFSAT_L64_KMIN, AFSAT_MAX_LEN, 4, 1, true, AFSAT_L64_THREADS, 1>(const EvalParams<double>);
template __global__ void k_eval_split<double, AFSAT_L64_KMIN, AFSAT_MAX_LEN, 4, 1, false, AFSAT_L64_THREADS, 1>(const EvalParams<double>);
#endif
#if AFSAT_M32_PACKED
template __global__ void k_eval_split<float, 9, AFSAT_B_KMAX32, 2, 2, true, AFSAT_M32_THREADS, 1>(const EvalParams<float>);
template __global__ void k_eval_split<float, 9, AFSAT_B_KMAX32, 2, 2, false, AFSAT_M32_THREADS, 1>(const EvalParams<float>);
#endif
}  // namespace afsat
