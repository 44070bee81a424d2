// afsat_ks32.cu -- the instantiations of the lane-split register kernels k_eval_split (SURVEY.md §8(a) a1-a5 for
// constraints longer than 8 literals in fp32 and 20 in fp64), in a translation unit of their own so
// that the per-length bodies compile in parallel with the rest of the build (build.py).
#define AFSAT_KS32_TU
#include "afsat_split.cuh"

namespace afsat {
template __global__ void k_eval_split<float, AFSAT_L32_KMIN, AFSAT_MAX_LEN, AFSAT_L32_NS, 1, true, AFSAT_L32_THREADS, AFSAT_L32_MINB>(const EvalParams<float>);
template __global__ void k_eval_split<float, AFSAT_L32_KMIN, AFSAT_MAX_LEN, AFSAT_L32_NS, 1, false, AFSAT_L32_THREADS, AFSAT_L32_MINB>(const EvalParams<float>);
template __global__ void k_eval_split<double, AFSAT_L64_KMIN, AFSAT_MAX_LEN, 4, 1, true, AFSAT_L64_THREADS, 1>(const EvalParams<double>);
template __global__ void k_eval_split<double, AFSAT_L64_KMIN, AFSAT_MAX_LEN, 4, 1, false, AFSAT_L64_THREADS, 1>(const EvalParams<double>);
template __global__ void k_eval_split<double, AFSAT_A_KMAX + 1, AFSAT_B_KMAX, 2, 1, true, AFSAT_L64_THREADS, 1>(const EvalParams<double>);
template __global__ void k_eval_split<double, AFSAT_A_KMAX + 1, AFSAT_B_KMAX, 2, 1, false, AFSAT_L64_THREADS, 1>(const EvalParams<double>);
template __global__ void k_eval_split<float, AFSAT_A_KMAX + 1, AFSAT_B_KMAX, 2, 2, true, AFSAT_M32_THREADS, AFSAT_M32_MINB>(const EvalParams<float>);
template __global__ void k_eval_split<float, AFSAT_A_KMAX + 1, AFSAT_B_KMAX, 2, 2, false, AFSAT_M32_THREADS, AFSAT_M32_MINB>(const EvalParams<float>);
}  // namespace afsat
