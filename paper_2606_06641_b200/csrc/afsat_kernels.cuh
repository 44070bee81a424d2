// afsat_kernels.cuh -- sm_100a device code of the AFSAT hot path.
//
// Mapping: LANE = CANDIDATE.  X is variable-major [n][ldb], so the k literal
// gathers of a constraint are k coalesced 128-byte row segments per warp, the constraint's
// literal list / signature / weight rows are warp-uniform (no divergence), and all prefix
// products live in registers.  A CTA covers one chunk of constraints of one length bucket
// (blockIdx.x -> work item) times 32*warps candidates (blockIdx.y).
//
// Per constraint and DFT point p the thread evaluates (afsat.h afsat_host_tables)
//     f_i = a_p + b_p y_i,  P = prod_i f_i,  FE += Re(w_p P),
//     dFE/dy_i += Re( (w_p b_p) * prefix_{i-1} * suffix_{i+1} )        (leave-one-out, no division)
// and scatter-adds s_i dFE/dy_i into G[v_i][b] with one coalesced RED per literal per warp.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace afsat {

constexpr int32_t LIT_NEG   = (int32_t)0x80000000u;  // y = -x (or the constant -1 when fixed)
constexpr int32_t LIT_FIXED = 0x40000000;            // y is the constant +-1, no gradient
constexpr int32_t LIT_VAR   = 0x3FFFFFFF;

struct SigDev {                 // 32 bytes, one per signature (type, k, param)
    int32_t row_off;            // first row in the weight table (8 scalars per row)
    int16_t n_real, n_cplx;     // real rows first, then complex rows
    uint64_t sat_lo, sat_hi;    // bit tau: satisfied with tau true literals
    int64_t pad;
};

struct Item {                   // one CTA-sized chunk of constraints of a single length k
    int32_t k;
    int32_t c_begin, c_end;     // constraint range in bucket order
    int32_t pad;
    int64_t lit_base;           // offset of c_begin's first packed literal
};

template <typename T>
struct EvalParams {
    const T *x;                 // [n][ldb]
    T *G;                       // [n][ldb] accumulated with RED (must be zero on entry) or null
    T *Fpart;                   // [n_items][ldb] per-item partial objective or null
    int32_t *satacc;            // [ldb] satisfied-count accumulator (RED.ADD.S32) or null
    const int32_t *lits;        // packed literals, bucket order
    const int32_t *cons_sig;    // signature id per constraint, bucket order
    const SigDev *sigs;
    const T *rows;              // weight table
    const Item *items;          // items of this launch
    int32_t item_index_base;    // row of Fpart for items[0]
    int32_t B;
    int64_t ldb;
};

template <typename T> __device__ __forceinline__ T fma_(T a, T b, T c);
template <> __device__ __forceinline__ float fma_<float>(float a, float b, float c) { return fmaf(a, b, c); }
template <> __device__ __forceinline__ double fma_<double>(double a, double b, double c) { return fma(a, b, c); }

template <typename T> __device__ __forceinline__ void red_add(T *p, T v) { atomicAdd(p, v); }

// ---- literal gather (a1) + sign rounding and count (a7, a8) --------------------------------
template <typename T>
__device__ __forceinline__ T gather_literal(const T *__restrict__ x, int64_t ldb, int64_t b, int32_t lit)
{
    T v;
    if (lit & LIT_FIXED) v = T(1);                                   // warp-uniform branch
    else v = x[(int64_t)(lit & LIT_VAR) * ldb + b];
    return (lit < 0) ? -v : v;
}

// a7: the VARIABLE rounds to True iff x < 0 (x = 0, -0.0 -> False); a negated literal is true iff
// the variable is False -- so the tie x = 0 makes the literal -x TRUE (y = -0.0 is not "< 0").
template <typename T>
__device__ __forceinline__ int literal_true(T y, int32_t lit)
{
    return (lit < 0) ? !(y > T(0)) : (y < T(0));      // y = -x for negated literals: x < 0 <=> y > 0
}

__device__ __forceinline__ int sat_bit(const SigDev &sg, int tau)
{
    return (int)(((tau < 64) ? (sg.sat_lo >> tau) : (sg.sat_hi >> (tau - 64))) & 1ull);
}

// ---- a2-a4 for one constraint of compile-time length K, everything in registers -------------
template <typename T, int K, bool GRAD, bool STORE_F>
__device__ __forceinline__ void eval_points_reg(const T (&y)[K], const T *__restrict__ rows,
                                                int n_real, int n_cplx, T &fe, T (&g)[K])
{
    const T *r = rows;
    for (int p = 0; p < n_real; ++p, r += 8) {                       // self-conjugate points
        const T a = r[0], b = r[2], w = r[4], wb = r[6];
        T pre[K];
        T run = fma_(b, y[0], a);
        pre[0] = T(1);
#pragma unroll
        for (int i = 1; i < K; ++i) { pre[i] = run; run *= fma_(b, y[i], a); }
        fe = fma_(w, run, fe);
        if (GRAD) {
            T suf = wb;
#pragma unroll
            for (int i = K - 1; i >= 1; --i) { g[i] = fma_(pre[i], suf, g[i]); suf *= fma_(b, y[i], a); }
            g[0] += suf;
        }
    }
    for (int p = 0; p < n_cplx; ++p, r += 8) {                       // one of each conjugate pair
        const T ar = r[0], ai = r[1], br = r[2], bi = r[3], wr = r[4], wi = r[5];
        T pr[K], pi[K], fr[STORE_F ? K : 1], fi[STORE_F ? K : 1];
        T rr = fma_(br, y[0], ar), ri = fma_(bi, y[0], ai);
        pr[0] = T(1); pi[0] = T(0);
        if (STORE_F) { fr[0] = rr; fi[0] = ri; }
#pragma unroll
        for (int i = 1; i < K; ++i) {
            const T f_r = fma_(br, y[i], ar), f_i = fma_(bi, y[i], ai);
            if (STORE_F) { fr[i] = f_r; fi[i] = f_i; }
            pr[i] = rr; pi[i] = ri;
            const T nr = fma_(rr, f_r, -(ri * f_i));
            const T ni = fma_(rr, f_i, ri * f_r);
            rr = nr; ri = ni;
        }
        fe = fma_(wr, rr, fe);
        fe = fma_(-wi, ri, fe);
        if (GRAD) {
            T sr = r[6], si = r[7];                                   // suffix seeded with w b
#pragma unroll
            for (int i = K - 1; i >= 1; --i) {
                g[i] = fma_(pr[i], sr, g[i]);
                g[i] = fma_(-pi[i], si, g[i]);
                const T f_r = STORE_F ? fr[i] : fma_(br, y[i], ar);
                const T f_i = STORE_F ? fi[i] : fma_(bi, y[i], ai);
                const T nr = fma_(sr, f_r, -(si * f_i));
                const T ni = fma_(sr, f_i, si * f_r);
                sr = nr; si = ni;
            }
            g[0] += sr;                                               // prefix_0 = 1
        }
    }
}

template <typename T, int K, bool GRAD>
__device__ __forceinline__ void run_item_reg(const EvalParams<T> &p, const Item &it, int64_t b, int item_row)
{
    const bool live = b < p.B;
    T fe_acc = T(0);
    int sat = 0;
    const int32_t *L = p.lits + it.lit_base;
    for (int c = it.c_begin; c < it.c_end; ++c, L += K) {
        const SigDev sg = p.sigs[p.cons_sig[c]];
        int32_t lit[K];
        T y[K], g[K];
        int tau = 0;
#pragma unroll
        for (int i = 0; i < K; ++i) lit[i] = __ldg(L + i);
#pragma unroll
        for (int i = 0; i < K; ++i) {
            y[i] = gather_literal(p.x, p.ldb, b, lit[i]);
            tau += literal_true(y[i], lit[i]);
            g[i] = T(0);
        }
        sat += sat_bit(sg, tau);
        eval_points_reg<T, K, GRAD, (K <= 10)>(y, p.rows + (int64_t)sg.row_off * 8, sg.n_real, sg.n_cplx, fe_acc, g);
        if (GRAD && live) {
#pragma unroll
            for (int i = 0; i < K; ++i)
                if (!(lit[i] & LIT_FIXED))
                    red_add(p.G + (int64_t)(lit[i] & LIT_VAR) * p.ldb + b, (lit[i] < 0) ? -g[i] : g[i]);
        }
    }
    if (live) {
        if (p.Fpart) p.Fpart[(int64_t)item_row * p.ldb + b] = fe_acc;
        if (p.satacc) atomicAdd(p.satacc + b, sat);
    }
}

template <typename T, int K, int KHI, bool GRAD>
struct DispatchK {
    static __device__ __forceinline__ void go(const EvalParams<T> &p, const Item &it, int64_t b, int row)
    {
        if (it.k == K) run_item_reg<T, K, GRAD>(p, it, b, row);
        else DispatchK<T, K + 1, KHI, GRAD>::go(p, it, b, row);
    }
};
template <typename T, int KHI, bool GRAD>
struct DispatchK<T, KHI, KHI, GRAD> {
    static __device__ __forceinline__ void go(const EvalParams<T> &p, const Item &it, int64_t b, int row)
    {
        run_item_reg<T, KHI, GRAD>(p, it, b, row);
    }
};

// Register kernel for one class of lengths [KLO, KHI]; it.k is CTA-uniform.
template <typename T, int KLO, int KHI, bool GRAD>
__global__ void __launch_bounds__(256) k_eval_reg(const EvalParams<T> p)
{
    const Item it = p.items[blockIdx.x];
    const int64_t b = (int64_t)blockIdx.y * blockDim.x + threadIdx.x;
    if (b >= p.ldb) return;
    DispatchK<T, KLO, KHI, GRAD>::go(p, it, b, p.item_index_base + blockIdx.x);
}

// ---- generic kernel for long constraints (runtime k <= 64): prefix products staged in shared
// memory as [i][lane] columns (conflict-free), suffix running in registers ---------------------
template <typename T, bool GRAD>
__global__ void __launch_bounds__(256) k_eval_long(const EvalParams<T> p, int kmax)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const Item it = p.items[blockIdx.x];
    const int64_t b = (int64_t)blockIdx.y * blockDim.x + threadIdx.x;
    if (b >= p.ldb) return;                                   // whole warps only (ldb % 32 == 0)
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    T *sy = reinterpret_cast<T *>(smem_raw) + (size_t)warp * 4 * kmax * 32 + lane;
    T *spr = sy + (size_t)kmax * 32, *spi = spr + (size_t)kmax * 32, *sg = spi + (size_t)kmax * 32;
    const int k = it.k;
    const bool live = b < p.B;
    T fe_acc = T(0);
    int sat = 0;
    const int32_t *L = p.lits + it.lit_base;
    for (int c = it.c_begin; c < it.c_end; ++c, L += k) {
        const SigDev sgd = p.sigs[p.cons_sig[c]];
        int tau = 0;
        for (int i = 0; i < k; ++i) {
            const int32_t lit_i = __ldg(L + i);
            const T yi = gather_literal(p.x, p.ldb, b, lit_i);
            tau += literal_true(yi, lit_i);
            sy[i * 32] = yi;
            sg[i * 32] = T(0);
        }
        sat += sat_bit(sgd, tau);
        const T *r = p.rows + (int64_t)sgd.row_off * 8;
        for (int q = 0; q < sgd.n_real; ++q, r += 8) {
            const T a = r[0], bb = r[2], w = r[4], wb = r[6];
            T run = T(1);
            for (int i = 0; i < k; ++i) { spr[i * 32] = run; run *= fma_(bb, sy[i * 32], a); }
            fe_acc = fma_(w, run, fe_acc);
            if (GRAD) {
                T suf = wb;
                for (int i = k - 1; i >= 0; --i) {
                    sg[i * 32] = fma_(spr[i * 32], suf, sg[i * 32]);
                    suf *= fma_(bb, sy[i * 32], a);
                }
            }
        }
        for (int q = 0; q < sgd.n_cplx; ++q, r += 8) {
            const T ar = r[0], ai = r[1], br = r[2], bi = r[3], wr = r[4], wi = r[5];
            T rr = T(1), ri = T(0);
            for (int i = 0; i < k; ++i) {
                const T yi = sy[i * 32];
                const T f_r = fma_(br, yi, ar), f_i = fma_(bi, yi, ai);
                spr[i * 32] = rr; spi[i * 32] = ri;
                const T nr = fma_(rr, f_r, -(ri * f_i));
                const T ni = fma_(rr, f_i, ri * f_r);
                rr = nr; ri = ni;
            }
            fe_acc = fma_(wr, rr, fe_acc);
            fe_acc = fma_(-wi, ri, fe_acc);
            if (GRAD) {
                T sr = r[6], si = r[7];
                for (int i = k - 1; i >= 0; --i) {
                    const T yi = sy[i * 32];
                    T gi = sg[i * 32];
                    gi = fma_(spr[i * 32], sr, gi);
                    gi = fma_(-spi[i * 32], si, gi);
                    sg[i * 32] = gi;
                    const T f_r = fma_(br, yi, ar), f_i = fma_(bi, yi, ai);
                    const T nr = fma_(sr, f_r, -(si * f_i));
                    const T ni = fma_(sr, f_i, si * f_r);
                    sr = nr; si = ni;
                }
            }
        }
        if (GRAD && live) {
            for (int i = 0; i < k; ++i) {
                const int32_t lit = __ldg(L + i);
                if (!(lit & LIT_FIXED)) {
                    const T gi = sg[i * 32];
                    red_add(p.G + (int64_t)(lit & LIT_VAR) * p.ldb + b, (lit < 0) ? -gi : gi);
                }
            }
        }
    }
    if (live) {
        if (p.Fpart) p.Fpart[(int64_t)(p.item_index_base + blockIdx.x) * p.ldb + b] = fe_acc;
        if (p.satacc) atomicAdd(p.satacc + b, sat);
    }
}

// ---- integer-only check (a7, a8): no floating-point arithmetic beyond the sign test ----------
template <typename T>
__global__ void __launch_bounds__(256) k_check(const EvalParams<T> p)
{
    const Item it = p.items[blockIdx.x];
    const int64_t b = (int64_t)blockIdx.y * blockDim.x + threadIdx.x;
    if (b >= p.B) return;
    const int k = it.k;
    int sat = 0;
    const int32_t *L = p.lits + it.lit_base;
    for (int c = it.c_begin; c < it.c_end; ++c, L += k) {
        const SigDev sg = p.sigs[p.cons_sig[c]];
        int tau = 0;
        for (int i = 0; i < k; ++i) {
            const int32_t lit_i = __ldg(L + i);
            tau += literal_true(gather_literal(p.x, p.ldb, b, lit_i), lit_i);
        }
        sat += sat_bit(sg, tau);
    }
    atomicAdd(p.satacc + b, sat);
}

// ---- F[b] = sum over items of Fpart[item][b], fixed order, accumulated in double ------------
template <typename T>
__global__ void k_reduce_F(const T *__restrict__ Fpart, int n_items, int64_t ldb, int B, T *__restrict__ F)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B) return;
    double s = 0.0;
    for (int i = 0; i < n_items; ++i) s += (double)Fpart[(int64_t)i * ldb + b];
    F[b] = (T)s;
}

// ---- per-candidate state machine of Alg. 1 (a8, a9) -----------------------------------------
// mode 0 (inside the loop, step t >= 2): satacc holds the count on X(t-1); newly solved candidates
//        get first_step = step_base + t - 1 and freeze.  mode 1 (tail): count on the final X(T).
__global__ void k_flags(int32_t *__restrict__ satacc, int B, int m, int mode, int step_value, int n_steps,
                        int32_t *__restrict__ sat_count, uint8_t *__restrict__ is_solution,
                        int32_t *__restrict__ first_step, int32_t *__restrict__ d_any, volatile int32_t *h_any)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B) return;
    const int s = satacc[b];
    satacc[b] = 0;
    if (mode == 1) sat_count[b] = s;
    if ((mode == 0 || n_steps >= 1) && s == m && !is_solution[b]) {
        is_solution[b] = 1;
        first_step[b] = step_value;
        if (atomicCAS(d_any, 0, 1) == 0) {
            d_any[1] = step_value;
            if (h_any) { h_any[1] = step_value; __threadfence_system(); h_any[0] = 1; }
        }
    }
}

// afsat_check epilogue: counts out, is_solution = (count == m), accumulator reset.
__global__ void k_check_finish(int32_t *__restrict__ satacc, int B, int m, int32_t *__restrict__ sat_count,
                               uint8_t *__restrict__ is_solution)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B) return;
    const int s = satacc[b];
    satacc[b] = 0;
    sat_count[b] = s;
    is_solution[b] = (uint8_t)(s == m);
}

__global__ void k_reset_state(int B, uint8_t *is_solution, int32_t *first_step)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b < B) { is_solution[b] = 0; first_step[b] = -1; }
}

// ---- projected step (a6) + freeze (a9) + gradient reset, elementwise over [n][ldb] ----------
template <typename T>
__global__ void __launch_bounds__(256) k_update(T *__restrict__ x, T *__restrict__ G, const int8_t *__restrict__ fixed,
                                               const uint8_t *__restrict__ is_solution, T eta, int n, int B, int64_t ldb)
{
    const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= ldb) return;
    const bool upd = (b < B) && !is_solution[b];
    for (int v = blockIdx.y; v < n; v += gridDim.y) {
        const int64_t idx = (int64_t)v * ldb + b;
        const T g = G[idx];
        G[idx] = T(0);
        if (upd && !fixed[v]) {
            T nx = fma_(-eta, g, x[idx]);
            nx = nx > T(1) ? T(1) : nx;
            nx = nx < T(-1) ? T(-1) : nx;
            x[idx] = nx;
        }
    }
}

}  // namespace afsat
