// afsat_step.cuh -- the non-evaluation kernels of the path: projected step, sign rounding,
// exact discrete count, per-candidate state, line-search bookkeeping, restarts; plus the ONE-LAUNCH step loop for
// small instances (k_step_small) and the FP-pipe peak probes.  Included by afsat.cu only.
#pragma once
#include "afsat_kernels.cuh"

namespace afsat {

// ---- a7: sign rounding as one bit per (variable, candidate): bits[v][b / 32] bit (b % 32) = (x < 0)
template <typename T>
__global__ void __launch_bounds__(CTA_THREADS) k_pack_signs(const T *__restrict__ x, uint32_t *__restrict__ bits, int n,
                                                           int B, int64_t ldb)
{
    const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= ldb) return;                                             // whole warps (ldb % 32 == 0)
    const int64_t ldw = ldb >> 5;
    for (int v = blockIdx.y; v < n; v += gridDim.y) {
        const bool t = (b < B) && (x[(int64_t)v * ldb + b] < T(0));   // True iff x < 0 (0, -0.0 -> False)
        const uint32_t w = __ballot_sync(0xffffffffu, t);
        if ((threadIdx.x & 31) == 0) bits[(int64_t)v * ldw + (b >> 5)] = w;
    }
}

// ---- a6 + a7 + a9: projected step on the candidate tile [b_begin, b_end), gradient scratch reset, sign bits of the
// NEW x.  Frozen (solved) candidates and fixed variables keep their x.  A thread owns VW = 16 / sizeof(T) ADJACENT
// candidates (one 16-byte load / store per array and row), tpr threads span a row of the tile, a CTA pass covers
// CTA_THREADS / tpr rows and every thread keeps UPD_UNROLL rows in flight.  The sign bits of a 32-candidate word come
// from the 32 / VW lanes that hold it (one REDUX.OR).
// rows in flight per thread / CTAs per SM of k_update (cfg4, ms of update per step: 4 / 8: 2.52, 8 / 8: 3.10, 8 / 4: 2.92,
// 1 / 64: 2.47, 2 / 16: 2.28)
#define AFSAT_UPD_UNROLL 2
#define AFSAT_UPD_CTAS_PER_SM 16
constexpr int UPD_UNROLL = AFSAT_UPD_UNROLL;
template <typename T> struct Vec16;
template <> struct Vec16<float>  { typedef float4 type;  static constexpr int VW = 4; };
template <> struct Vec16<double> { typedef double2 type; static constexpr int VW = 2; };
__device__ __forceinline__ void vec_get(const float4 &v, float (&a)[4]) { a[0] = v.x; a[1] = v.y; a[2] = v.z; a[3] = v.w; }
__device__ __forceinline__ void vec_get(const double2 &v, double (&a)[2]) { a[0] = v.x; a[1] = v.y; }
__device__ __forceinline__ float4 vec_make(const float (&a)[4]) { return make_float4(a[0], a[1], a[2], a[3]); }
__device__ __forceinline__ double2 vec_make(const double (&a)[2]) { return make_double2(a[0], a[1]); }

template <typename T>
__global__ void __launch_bounds__(CTA_THREADS) k_update(T *__restrict__ x, T *__restrict__ G, int64_t g_ld, int64_t g_b0,
                                                       const int8_t *__restrict__ fixed,
                                                       const uint8_t *__restrict__ is_solution, uint32_t *__restrict__ bits,
                                                       T eta, int n, int B, int64_t ldb, int64_t b_begin, int64_t b_end,
                                                       int tpr)
{
    typedef typename Vec16<T>::type VT;
    constexpr int VW = Vec16<T>::VW, LPW = 32 / VW;                   // lanes per 32-candidate word
    const int col = threadIdx.x % tpr, r = threadIdx.x / tpr, rows_per_pass = blockDim.x / tpr;
    const int64_t b = b_begin + ((int64_t)blockIdx.x * tpr + col) * VW;
    if (b >= b_end) return;                                           // tiles are multiples of 32 candidates: whole word groups
    bool live[VW], upd[VW], any_upd = false;
#pragma unroll
    for (int j = 0; j < VW; ++j) {
        live[j] = b + j < B;
        upd[j] = live[j] && !is_solution[b + j];
        any_upd |= upd[j];
    }
    const int lane = threadIdx.x & 31;
    const unsigned wmask = ((LPW == 32) ? 0xffffffffu : ((1u << LPW) - 1u)) << (lane / LPW * LPW);
    const int sh = (lane % LPW) * VW;
    const int64_t ldw = ldb >> 5;
    const int stride = gridDim.y * rows_per_pass;
    for (int v0 = blockIdx.y * rows_per_pass + r; v0 < n; v0 += stride * UPD_UNROLL) {
        VT g[UPD_UNROLL], xv[UPD_UNROLL];
        int8_t fx[UPD_UNROLL];
#pragma unroll
        for (int u = 0; u < UPD_UNROLL; ++u) {
            const int v = v0 + u * stride;
            if (v < n) {
                g[u] = *reinterpret_cast<const VT *>(G + (int64_t)v * g_ld + (b - g_b0));
                xv[u] = __ldcs(reinterpret_cast<const VT *>(x + (int64_t)v * ldb + b));   // X streams through (evict-first): it is not
                                                                                          // needed again before the next step, and the
                                                                                          // gradient scratch stays in the L2 instead
                fx[u] = fixed[v];
            }
        }
#pragma unroll
        for (int u = 0; u < UPD_UNROLL; ++u) {
            const int v = v0 + u * stride;
            if (v < n) {                                              // uniform over the lanes of a word (same row)
                T gv[VW], xs[VW];
                vec_get(g[u], gv); vec_get(xv[u], xs);
                T zero[VW];
#pragma unroll
                for (int j = 0; j < VW; ++j) zero[j] = T(0);
                *reinterpret_cast<VT *>(G + (int64_t)v * g_ld + (b - g_b0)) = vec_make(zero);
                uint32_t nib = 0u;
#pragma unroll
                for (int j = 0; j < VW; ++j) {
                    T nx = xs[j];
                    if (upd[j] && !fx[u]) {
                        nx = fma_(-eta, gv[j], nx);
                        nx = nx > T(1) ? T(1) : nx;
                        nx = nx < T(-1) ? T(-1) : nx;
                    }
                    xs[j] = nx;
                    nib |= (uint32_t)(live[j] && (nx < T(0))) << j;
                }
                if (any_upd && !fx[u]) __stcs(reinterpret_cast<VT *>(x + (int64_t)v * ldb + b), vec_make(xs));
                const uint32_t w = __reduce_or_sync(wmask, nib << sh);
                if (lane % LPW == 0) bits[(int64_t)v * ldw + (b >> 5)] = w;
            }
        }
    }
}

// ---- a8: exact discrete count, integer only.  One thread = one 32-candidate word; the number tau
// of true literals is kept BIT-SLICED (t[j] holds bit j of tau for 32 candidates), the predicate is
// evaluated by scanning the smaller of {satisfied counts, violated counts}, and the per-candidate
// number of satisfied constraints of the item is again a bit-sliced counter.  The bit rows of a constraint's
// literals are requested CHK_MLP at a time before any is consumed (the kernel is bound by the latency of those loads).
struct CheckParams {
    const uint32_t *bits;       // [n][ldw]
    int64_t ldw;
    const int32_t *lits;
    const SigDev *sigs;
    const Item *items;
    int32_t *satacc;            // [ldb]
    int32_t B;
    int32_t w_begin, w_end;     // word range of this launch
    int32_t wpb;                // words per CTA (power of two <= 32)
    int32_t n_items;
    int32_t *step_ctr;          // or null: incremented once per launch (the step index of a replayed CUDA graph)
};
constexpr int CHK_MLP = 8;
// SigDev::chk_kind: predicates of the count tau of true literals that need no counting
enum { CHK_GENERAL = 0, CHK_OR = 1 /* tau >= 1 */, CHK_NONE = 2 /* tau == 0 */, CHK_ALL = 3 /* tau == k */,
       CHK_NAND = 4 /* tau < k */, CHK_NAE = 5 /* 0 < tau < k */, CHK_EQ = 6 /* tau in {0, k} */, CHK_ODD = 7, CHK_EVEN = 8 };

// satisfied-mask of ONE constraint for the 32 candidates of a word.  bw: the word's column of the sign-bit array; the bit
// rows of up to MLP literals are requested before any is consumed.
template <int MLP>
__device__ __forceinline__ uint32_t chk_constraint(const int32_t *__restrict__ L, int k, const uint32_t *__restrict__ bw, uint32_t ldw,
                                                   int kind, int nb, uint64_t scan_lo, uint64_t scan_hi, int scan_is_sat)
{
    if (kind != CHK_GENERAL) {
        // predicates that are a function of (any literal true, all literals true, parity): no counting at all
        uint32_t any = 0u, all = 0xffffffffu, par = 0u;
        for (int i0 = 0; i0 < k; i0 += MLP) {
            uint32_t mm[MLP];
#pragma unroll
            for (int u = 0; u < MLP; ++u)
                if (i0 + u < k) {
                    const int32_t lit = L[i0 + u];
                    const uint32_t w = __ldg(bw + (size_t)(uint32_t)(lit & LIT_VAR) * ldw);
                    mm[u] = lit < 0 ? ~w : w;                         // literal true = variable true XOR negated
                }
#pragma unroll
            for (int u = 0; u < MLP; ++u)
                if (i0 + u < k) { any |= mm[u]; all &= mm[u]; par ^= mm[u]; }
        }
        return kind == CHK_OR ? any : kind == CHK_NONE ? ~any : kind == CHK_ALL ? all : kind == CHK_NAND ? ~all
             : kind == CHK_NAE ? (any & ~all) : kind == CHK_EQ ? (all | ~any) : kind == CHK_ODD ? par : ~par;
    }
    uint32_t t[7] = {0u, 0u, 0u, 0u, 0u, 0u, 0u};                     // tau, bit-sliced
    for (int i0 = 0; i0 < k; i0 += MLP) {
        uint32_t mm[MLP];
#pragma unroll
        for (int u = 0; u < MLP; ++u)
            if (i0 + u < k) {
                const int32_t lit = L[i0 + u];
                const uint32_t w = __ldg(bw + (size_t)(uint32_t)(lit & LIT_VAR) * ldw);
                mm[u] = lit < 0 ? ~w : w;
            }
#pragma unroll
        for (int u = 0; u < MLP; ++u)
            if (i0 + u < k) {
                uint32_t m = mm[u];
#pragma unroll
                for (int j = 0; j < 7; ++j)
                    if (j < nb) { const uint32_t sv = t[j] ^ m; m &= t[j]; t[j] = sv; }
            }
    }
    uint32_t acc = 0u;
    for (int tau = 0; tau <= k; ++tau) {
        const uint64_t bit = tau < 64 ? (scan_lo >> tau) : (scan_hi >> (tau - 64));
        if (!(bit & 1ull)) continue;
        uint32_t eq = 0xffffffffu;
#pragma unroll
        for (int j = 0; j < 7; ++j)
            if (j < nb) eq &= ((tau >> j) & 1) ? t[j] : ~t[j];
        acc |= eq;
    }
    return scan_is_sat ? acc : ~acc;                                  // 1 = constraint satisfied
}

// The constraints [grp, nc) step ngrp of an item whose predicate needs no count, with the length and the combination known at
// compile time (MODE 0: any literal true, 1: all true, 2: any and not all, 3: parity; inv flips the result: NONE, NAND, EQ,
// EVEN).  s_var / s_neg: the item's literals as staged by the CTA -- variable, and 0 / ~0 for a negated literal.  All K bit
// rows are requested before any is consumed; ~9 instructions per literal against ~30 of the general routine.
template <int K, int MODE, typename Tally>
__device__ __forceinline__ void chk_item_simple(const int32_t *__restrict__ s_var, const uint32_t *__restrict__ s_neg, int nc, int grp,
                                                int ngrp, const uint32_t *__restrict__ bw, uint32_t ldw, uint32_t inv, Tally &&tally)
{
    for (int c = grp; c < nc; c += ngrp) {
        uint32_t mm[K];
#pragma unroll
        for (int i = 0; i < K; ++i) mm[i] = __ldg(bw + (size_t)(uint32_t)s_var[c * K + i] * ldw);
        uint32_t any = 0u, all = 0xffffffffu, par = 0u;
#pragma unroll
        for (int i = 0; i < K; ++i) {
            const uint32_t m = mm[i] ^ s_neg[c * K + i];              // literal true = variable true XOR negated
            if (MODE == 0 || MODE == 2) any |= m;
            if (MODE == 1 || MODE == 2) all &= m;
            if (MODE == 3) par ^= m;
        }
        tally((MODE == 0 ? any : MODE == 1 ? all : MODE == 2 ? (any & ~all) : par) ^ inv);
    }
}

template <int MODE, typename Tally>
__device__ __forceinline__ void chk_item_simple_k(int k, const int32_t *s_var, const uint32_t *s_neg, int nc, int grp, int ngrp,
                                                  const uint32_t *bw, uint32_t ldw, uint32_t inv, Tally &&tally)
{
    switch (k) {
    case 1: chk_item_simple<1, MODE>(s_var, s_neg, nc, grp, ngrp, bw, ldw, inv, tally); break;
    case 2: chk_item_simple<2, MODE>(s_var, s_neg, nc, grp, ngrp, bw, ldw, inv, tally); break;
    case 3: chk_item_simple<3, MODE>(s_var, s_neg, nc, grp, ngrp, bw, ldw, inv, tally); break;
    case 4: chk_item_simple<4, MODE>(s_var, s_neg, nc, grp, ngrp, bw, ldw, inv, tally); break;
    case 5: chk_item_simple<5, MODE>(s_var, s_neg, nc, grp, ngrp, bw, ldw, inv, tally); break;
    case 6: chk_item_simple<6, MODE>(s_var, s_neg, nc, grp, ngrp, bw, ldw, inv, tally); break;
    case 7: chk_item_simple<7, MODE>(s_var, s_neg, nc, grp, ngrp, bw, ldw, inv, tally); break;
    default: chk_item_simple<8, MODE>(s_var, s_neg, nc, grp, ngrp, bw, ldw, inv, tally); break;
    }
}

__global__ void __launch_bounds__(CTA_THREADS, 4) k_check_bits(const CheckParams p)
{
    __shared__ int32_t s_lits[LIT_CHUNK];
    __shared__ uint32_t s_neg[LIT_CHUNK];                             // short simple items: 0 / ~0 per literal (s_lits then holds the variable)
    __shared__ int32_t s_cnt[32 * 32];
    if (p.step_ctr && blockIdx.x == 0 && blockIdx.y == 0 && threadIdx.x == 0) ++p.step_ctr[0];
    const int wpb = p.wpb, n_items = p.n_items;
    const uint32_t ldw = (uint32_t)p.ldw;
    for (int i = threadIdx.x; i < wpb * 32; i += blockDim.x) s_cnt[i] = 0;
    const int wi = threadIdx.x % wpb, grp = threadIdx.x / wpb, ngrp = blockDim.x / wpb;
    const int word = p.w_begin + blockIdx.y * wpb + wi;
    const bool valid = word < p.w_end;
    const uint32_t *bw = p.bits + (valid ? word : p.w_begin);
    const Item *items = p.items;
    const SigDev *sigs = p.sigs;
    const int32_t *lits = p.lits;
    // satisfied constraints per candidate, bit-sliced, in two levels: a 3-plane counter takes 7 constraints, then it is
    // added into the 13-plane counter (a full 13-plane ripple per constraint was a third of this kernel's instructions)
    uint32_t cnt[13], lo[3] = {0u, 0u, 0u};
#pragma unroll
    for (int j = 0; j < 13; ++j) cnt[j] = 0u;
    int nlo = 0, nacc = 0;                                            // constraints in lo[] / in cnt[] + lo[] so far
    auto fold = [&]() {                                               // cnt += lo (3-plane value), lo = 0
        uint32_t carry = 0u;
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            const uint32_t a = cnt[j], bq = lo[j];
            cnt[j] = a ^ bq ^ carry;
            carry = (a & bq) | (carry & (a ^ bq));
            lo[j] = 0u;
        }
#pragma unroll
        for (int j = 3; j < 13; ++j) { const uint32_t sv = cnt[j] ^ carry; carry &= cnt[j]; cnt[j] = sv; }
        nlo = 0;
    };
    auto flush = [&]() {                                              // bit-sliced counter -> per-candidate integers
        fold();
        for (int bit = 0; bit < 32; ++bit) {
            int val = 0;
#pragma unroll
            for (int j = 0; j < 13; ++j) val |= (int)((cnt[j] >> bit) & 1u) << j;
            if (val) atomicAdd(&s_cnt[wi * 32 + bit], val);
        }
#pragma unroll
        for (int j = 0; j < 13; ++j) cnt[j] = 0u;
        nacc = 0;
    };
    for (int item = blockIdx.x; item < n_items; item += gridDim.x) {  // persistent over work items
        const Item it = items[item];
        const SigDev sg = sigs[it.sig];
        const int k = it.k, nc = it.c_end - it.c_begin, kind = sg.chk_kind, sis = sg.scan_is_sat;
        const uint64_t slo = sg.scan_lo, shi = sg.scan_hi;
        const bool simple = kind != CHK_GENERAL && k <= 8;            // (CTA-uniform)
        __syncthreads();                                              // previous item's literals are consumed
        for (int i = threadIdx.x; i < nc * k; i += blockDim.x) {
            const int32_t l = __ldg(lits + it.lit_base + i);
            s_lits[i] = simple ? (l & LIT_VAR) : l;
            if (simple) s_neg[i] = l < 0 ? 0xffffffffu : 0u;
        }
        __syncthreads();
        if (!valid) continue;
        int nb = 1;
        while ((1 << nb) <= k) ++nb;                                  // bits of tau in [0, k]
        const int mine = (nc - grp + ngrp - 1) / ngrp;
        if (nacc + mine > 8000) flush();
        nacc += mine > 0 ? mine : 0;
        auto tally = [&](uint32_t carry) {                            // one more constraint's satisfied-mask into the counter
#pragma unroll
            for (int j = 0; j < 3; ++j) { const uint32_t sv = lo[j] ^ carry; carry &= lo[j]; lo[j] = sv; }
            if (++nlo == 7) fold();
        };
        if (simple) {
            const uint32_t inv = (kind == CHK_NONE || kind == CHK_NAND || kind == CHK_EQ || kind == CHK_EVEN) ? 0xffffffffu : 0u;
            if (kind == CHK_OR || kind == CHK_NONE) chk_item_simple_k<0>(k, s_lits, s_neg, nc, grp, ngrp, bw, ldw, inv, tally);
            else if (kind == CHK_ALL || kind == CHK_NAND) chk_item_simple_k<1>(k, s_lits, s_neg, nc, grp, ngrp, bw, ldw, inv, tally);
            else if (kind == CHK_NAE || kind == CHK_EQ) chk_item_simple_k<2>(k, s_lits, s_neg, nc, grp, ngrp, bw, ldw, inv, tally);
            else chk_item_simple_k<3>(k, s_lits, s_neg, nc, grp, ngrp, bw, ldw, inv, tally);
            continue;
        }
        for (int c = grp; c < nc; c += ngrp) {
            const int32_t *L = s_lits + c * k;
            tally(k <= 4 ? chk_constraint<4>(L, k, bw, ldw, kind, nb, slo, shi, sis)
                         : chk_constraint<8>(L, k, bw, ldw, kind, nb, slo, shi, sis));
        }
    }
    if (valid && nacc) flush();
    __syncthreads();
    const int64_t b0 = ((int64_t)p.w_begin + (int64_t)blockIdx.y * wpb) * 32;
    for (int i = threadIdx.x; i < wpb * 32; i += blockDim.x) {
        const int64_t b = b0 + i;
        if (b < p.B && b < (int64_t)p.w_end * 32 && s_cnt[i]) atomicAdd(p.satacc + b, s_cnt[i]);
    }
}

// ---- line search (afsat_step_ls; reading B5): per-candidate backtracking along the projection arc ----
// ls_state[b]: 0 = still searching, 1 = step accepted, 2 = frozen (solved or converged)
constexpr int LS_CHUNKS = 32;         // row chunks of the <G, X - X'> reduction (fixed-order two-stage sum)

__global__ void k_ls_begin(int B, int64_t ldb, const uint8_t *__restrict__ is_solution, const uint8_t *__restrict__ converged,
                           uint8_t *__restrict__ ls_state, double s_max, double *__restrict__ eta)
{
    const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= ldb) return;
    ls_state[b] = (b >= B || is_solution[b] || converged[b]) ? 2 : 0;
    eta[b] = s_max;
}

// the partial assignment of candidate b: fixed[(b / group_w) * n + v]  (several partial assignments)
__device__ __forceinline__ const int8_t *fixed_of(const int8_t *fixed, int64_t b, int64_t group_w, int n_groups, int n)
{
    int64_t g = b / group_w;
    if (g >= n_groups) g = n_groups - 1;
    return fixed + g * (int64_t)n;
}

// X' = clamp(X - eta_b G) for the candidates still searching (first trial: every candidate gets a valid X'),
// Dpart[chunk][b] = sum over the chunk's rows of G (X - X')
template <typename T>
__global__ void __launch_bounds__(CTA_THREADS) k_ls_trial(const T *__restrict__ x, const T *__restrict__ G, T *__restrict__ xt,
                                                         const int8_t *__restrict__ fixed_all, int64_t group_w, int n_groups,
                                                         const uint8_t *__restrict__ ls_state,
                                                         const double *__restrict__ eta, double *__restrict__ Dpart, int n,
                                                         int64_t ldb, int first_trial)
{
    const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= ldb) return;
    const int st = ls_state[b];
    const int rows = (n + LS_CHUNKS - 1) / LS_CHUNKS, v0 = blockIdx.y * rows, v1 = min(n, v0 + rows);
    if (st != 0) {
        if (first_trial) for (int v = v0; v < v1; ++v) xt[(int64_t)v * ldb + b] = x[(int64_t)v * ldb + b];
        return;
    }
    const int8_t *fixed = fixed_of(fixed_all, b, group_w, n_groups, n);
    const T e = (T)eta[b];
    double D = 0.0;
    for (int v = v0; v < v1; ++v) {
        const T xv = x[(int64_t)v * ldb + b];
        T nx = xv;
        if (!fixed[v]) {
            const T g = G[(int64_t)v * ldb + b];
            nx = fma_(-e, g, xv);
            nx = nx > T(1) ? T(1) : nx;
            nx = nx < T(-1) ? T(-1) : nx;
            D += (double)g * (double)(xv - nx);
        }
        xt[(int64_t)v * ldb + b] = nx;
    }
    Dpart[(int64_t)blockIdx.y * ldb + b] = D;
}

// Armijo test of the trial; backtrack or give up (eta < delta: converged)
template <typename T>
__global__ void k_ls_decide(int B, int64_t ldb, const T *__restrict__ F0, const T *__restrict__ F1, const double *__restrict__ Dpart,
                            uint8_t *__restrict__ ls_state, double *__restrict__ eta, uint8_t *__restrict__ converged, double c1,
                            double beta, double delta)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B || ls_state[b] != 0) return;
    double D = 0.0;
    for (int c = 0; c < LS_CHUNKS; ++c) D += Dpart[(int64_t)c * ldb + b];
    if ((double)F1[b] <= (double)F0[b] - c1 * D) { ls_state[b] = 1; return; }
    const double e = eta[b] * beta;
    eta[b] = e;
    if (e < delta) { ls_state[b] = 2; converged[b] = 1; }
}

// accepted candidates take X', sign bits of the resulting X for everyone
template <typename T>
__global__ void __launch_bounds__(CTA_THREADS) k_ls_commit(T *__restrict__ x, const T *__restrict__ xt, const uint8_t *__restrict__ ls_state,
                                                          uint32_t *__restrict__ bits, int n, int B, int64_t ldb)
{
    const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= ldb) return;                                             // whole warps (ldb % 32 == 0)
    const bool live = b < B, take = live && ls_state[b] == 1;
    const int64_t ldw = ldb >> 5;
    for (int v = blockIdx.y; v < n; v += gridDim.y) {
        T xv = T(0);
        if (live) {
            xv = take ? xt[(int64_t)v * ldb + b] : x[(int64_t)v * ldb + b];
            if (take) x[(int64_t)v * ldb + b] = xv;
        }
        const uint32_t w = __ballot_sync(0xffffffffu, live && xv < T(0));
        if ((threadIdx.x & 31) == 0) bits[(int64_t)v * ldw + (b >> 5)] = w;
    }
}

template <typename T>
__global__ void k_ls_report(int B, const double *__restrict__ eta, T *__restrict__ eta_out)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b < B) eta_out[b] = (T)eta[b];
}

// ---- afsat_restart: counter-based uniform re-initialisation (include/afsat.h states the generator) ----
__device__ __forceinline__ uint32_t fmix32(uint32_t h)
{
    h ^= h >> 16; h *= 0x85EBCA6Bu; h ^= h >> 13; h *= 0xC2B2AE35u; h ^= h >> 16;
    return h;
}

template <typename T>
__global__ void __launch_bounds__(CTA_THREADS) k_restart(T *__restrict__ x, const int8_t *__restrict__ fixed_all, int64_t group_w,
                                                        int n_groups, const uint8_t *__restrict__ keep, uint32_t lo, uint32_t hi,
                                                        uint32_t round, int n, int B, int64_t ldb)
{
    const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B || (keep && keep[b])) return;
    const int8_t *fixed = fixed_of(fixed_all, b, group_w, n_groups, n);
    const uint32_t hb = fmix32(lo ^ ((uint32_t)b * 0x9E3779B9u));
    for (int v = blockIdx.y; v < n; v += gridDim.y) {
        const int8_t f = fixed[v];
        T val;
        if (f) val = (T)f;
        else {
            const uint32_t h = fmix32(fmix32((hb + (uint32_t)v * 0x85EBCA6Bu) ^ hi) + round * 0xC2B2AE35u);
            val = (T)((float)(h >> 8) * 1.1920928955078125e-07f - 1.0f);     // (h >> 8) 2^-23 - 1, exact
        }
        x[(int64_t)v * ldb + b] = val;
    }
}

// zero the padding columns [B, ldb) of a caller-owned gradient (vector REDs of a lane pair that
// straddles B spill into them)
template <typename T>
__global__ void k_zero_pad(T *__restrict__ G, int n, int B, int64_t ldb)
{
    const int64_t np = ldb - B;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < (int64_t)n * np; i += (int64_t)gridDim.x * blockDim.x)
        G[(i / np) * ldb + B + (i % np)] = T(0);
}

// ---- F[b] = F_const + sum over items of Fpart[item][b], in a FIXED order, accumulated in double, for the candidates
// [b0, b1) of one partial-assignment group (F_const: the constraints the partial assignment already decides).
// A CTA takes 32 candidates; its RED_F_SLICES warps sum the rows i = slice, slice + RED_F_SLICES, ... (a thread per
// candidate walking all rows alone was latency-bound: 65 us on cfg3), then slice 0 adds the slices' sums in slice order.
constexpr int RED_F_SLICES = 16;
template <typename T>
__global__ void __launch_bounds__(32 * RED_F_SLICES) k_reduce_F(const T *__restrict__ Fpart, int n_rows, int64_t ldb, int64_t b0, int64_t b1,
                                                                double F_const, T *__restrict__ F, const uint8_t *__restrict__ skip)
{
    __shared__ double s_part[RED_F_SLICES][32];
    const int lane = threadIdx.x & 31, slice = threadIdx.x >> 5;
    const int64_t b = b0 + (int64_t)blockIdx.x * 32 + lane;
    const bool live = b < b1 && !(skip && skip[b]);                    // skipped candidates keep their F
    double s = 0.0;
    if (live) {
        const T *col = Fpart + b;
#pragma unroll 4
        for (int i = slice; i < n_rows; i += RED_F_SLICES) s += (double)col[(int64_t)i * ldb];
    }
    s_part[slice][lane] = s;
    __syncthreads();
    if (slice == 0 && live) {
        double t = F_const;
#pragma unroll
        for (int j = 0; j < RED_F_SLICES; ++j) t += s_part[j][lane];
        F[b] = (T)t;
    }
}

// ---- per-candidate state machine of Alg. 1 (a8, a9): satacc holds the count on the current X over the constraints
// that reach a kernel; sat_const[g] adds the ones group g's partial assignment satisfies outright ----
// d_any: {flag, first step, -, step counter}
__global__ void k_flags(int32_t *__restrict__ satacc, int B, int m, int mark_solved, int step_value, const int32_t *step_ctr,
                        const int32_t *__restrict__ sat_const, int64_t group_w, int n_groups,
                        int32_t *__restrict__ sat_count, uint8_t *__restrict__ is_solution,
                        int32_t *__restrict__ first_step, int32_t *__restrict__ d_any, volatile int32_t *h_any)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B) return;
    if (step_ctr) step_value = step_ctr[0];
    int64_t g = b / group_w;
    if (g >= n_groups) g = n_groups - 1;
    const int s = satacc[b] + sat_const[g];
    satacc[b] = 0;
    sat_count[b] = s;
    if (mark_solved && s == m && !is_solution[b]) {
        is_solution[b] = 1;
        first_step[b] = step_value;
        if (atomicCAS(d_any, 0, 1) == 0) {
            d_any[1] = step_value;
            if (h_any) { h_any[1] = step_value; __threadfence_system(); h_any[0] = 1; }
        }
    }
}

// afsat_check epilogue: counts out, is_solution = (count == m), accumulator reset.
__global__ void k_check_finish(int32_t *__restrict__ satacc, int B, int m, const int32_t *__restrict__ sat_const, int64_t group_w,
                               int n_groups, int32_t *__restrict__ sat_count, uint8_t *__restrict__ is_solution)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B) return;
    int64_t g = b / group_w;
    if (g >= n_groups) g = n_groups - 1;
    const int s = satacc[b] + sat_const[g];
    satacc[b] = 0;
    sat_count[b] = s;
    is_solution[b] = (uint8_t)(s == m);
}

// start of a step call, ON THE STREAM: per-candidate state (unless resuming), the any-solved flag on the device and
// in the caller's pinned host memory, the step counter of a replayed graph
__global__ void k_reset_state(int B, int reset_candidates, uint8_t *is_solution, int32_t *first_step, int32_t *d_any,
                              volatile int32_t *h_any, int step_base)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (reset_candidates && b < B) { is_solution[b] = 0; first_step[b] = -1; }
    if (b == 0) {
        d_any[0] = 0; d_any[1] = 0x7fffffff; d_any[2] = 0; d_any[3] = step_base;
        if (h_any) { h_any[0] = 0; h_any[1] = -1; }
    }
}

// ---- the whole step loop in ONE launch (small instances: PAPER.md:81 "compiled once and executed repeatedly", :103
// the lock-step loop runs on the accelerator) ------------------------------------------------
// Such instances are bound by launch latency, not by arithmetic (cfg0: 1.4e4 evaluations per step), and a batch of a
// few dozen candidates cannot fill the machine with lane = candidate.  So here a CTA owns ONE candidate for all n_steps
// iterations and its THREADS share out the constraints (thread = constraint; bucket order keeps the constraints of a
// warp on one signature, so the length switch rarely diverges): X and G of the candidate live in shared memory, partial
// gradients meet in shared-memory atomics, and the gather of iteration t + 1 also yields the signs of X(t), so the
// exact count (a8) rides on the same pass.  Candidates never exchange data: no CTA waits on another, and a solved
// candidate's CTA simply ends.  Lengths k <= 8 only (one register body per length).
struct ConsDev { int32_t lit_off; int16_t sig; int16_t k; };       // one constraint in bucket order

template <typename T>
struct SmallParams {
    T *x;                       // [n][ldb], in/out
    int64_t ldb;
    int32_t n, B, m, m_live;
    const int32_t *lits;
    const ConsDev *cons;
    const SigDev *sigs;
    const T *rows;
    const int8_t *fixed;
    T eta;
    int32_t n_steps, step_base, sat_const;
    int32_t *sat_count;
    uint8_t *is_solution;
    int32_t *first_step;
    int32_t *d_any;             // {flag, first step (min), finished CTAs, -}
    volatile int32_t *h_any;
};
constexpr int SMALL_THREADS = 512;

template <typename T, int K, bool GRAD>
__device__ __forceinline__ int small_constraint(const int32_t *__restrict__ L, const T *__restrict__ sx, T *__restrict__ sg,
                                                const T *__restrict__ tab, int n_real, int n_cplx, uint64_t scan_lo, int scan_is_sat)
{
    int32_t lit[K];
    T y[K][1], g[K][1], fe[1] = {T(0)};
    int tau = 0;
#pragma unroll
    for (int i = 0; i < K; ++i) lit[i] = __ldg(L + i);
#pragma unroll
    for (int i = 0; i < K; ++i) {
        const T xv = sx[lit[i] & LIT_VAR];
        tau += (int)((xv < T(0)) != (lit[i] < 0));                    // literal true = variable true XOR negated (B2)
        y[i][0] = flip_sign(xv, lit[i]);
        g[i][0] = T(0);
    }
    if (GRAD) {
        eval_points_reg<T, K, 1, true>(y, tab, n_real, n_cplx, fe, g);
#pragma unroll
        for (int i = 0; i < K; ++i) atomicAdd(sg + (lit[i] & LIT_VAR), flip_sign(g[i][0], lit[i]));
    }
    return (int)((scan_lo >> tau) & 1ull) == scan_is_sat;             // k <= 8: tau < 64
}

template <typename T>
__global__ void __launch_bounds__(SMALL_THREADS, 1) k_step_small(const SmallParams<T> p)
{
    extern __shared__ __align__(16) unsigned char s_raw[];
    T *sx = reinterpret_cast<T *>(s_raw), *sg = sx + p.n;
    __shared__ int s_cnt, s_frozen;
    const int t = threadIdx.x, nt = blockDim.x;
    const int64_t b = blockIdx.x;
    for (int v = t; v < p.n; v += nt) sx[v] = p.x[(int64_t)v * p.ldb + b];
    if (t == 0) { s_frozen = (int)p.is_solution[b]; s_cnt = 0; }
    int last = 0;
    for (int it = 0; it <= p.n_steps; ++it) {
        const bool grad = it < p.n_steps;
        if (grad) for (int v = t; v < p.n; v += nt) sg[v] = T(0);
        __syncthreads();
        if (s_frozen && it > 0) break;                                // solved: X and its count no longer change (a9)
        int cnt = 0;
        for (int j = t; j < p.m_live; j += nt) {
            const ConsDev c = p.cons[j];
            const int32_t *L = p.lits + c.lit_off;
            const SigDev *sd = p.sigs + c.sig;
            const T *tab = p.rows + (int64_t)sd->row_off * 8;
            const int n_real = sd->n_real, n_cplx = sd->n_cplx, sis = sd->scan_is_sat;
            const uint64_t slo = sd->scan_lo;
#define AFSAT_SMALL_CASE(K_) case K_: cnt += grad ? small_constraint<T, K_, true>(L, sx, sg, tab, n_real, n_cplx, slo, sis) \
                                                  : small_constraint<T, K_, false>(L, sx, sg, tab, n_real, n_cplx, slo, sis); break;
            switch (c.k) {
                AFSAT_SMALL_CASE(1) AFSAT_SMALL_CASE(2) AFSAT_SMALL_CASE(3) AFSAT_SMALL_CASE(4)
                AFSAT_SMALL_CASE(5) AFSAT_SMALL_CASE(6) AFSAT_SMALL_CASE(7) AFSAT_SMALL_CASE(8)
            }
#undef AFSAT_SMALL_CASE
        }
        cnt = __reduce_add_sync(0xffffffffu, cnt);
        if ((t & 31) == 0 && cnt) atomicAdd(&s_cnt, cnt);
        __syncthreads();
        if (t == 0) {                                                 // a8, a9 on X(it): X(0) is counted but not marked (A11)
            last = s_cnt + p.sat_const;
            s_cnt = 0;
            if (it >= 1 && last == p.m && !s_frozen) {
                s_frozen = 1;
                p.is_solution[b] = 1;
                const int step = p.step_base + it;
                p.first_step[b] = step;
                atomicExch(p.d_any, 1);
                const int prev = atomicMin(p.d_any + 1, step);
                if (p.h_any && step < prev) { p.h_any[1] = step; __threadfence_system(); p.h_any[0] = 1; }
            }
        }
        if (!grad) break;
        __syncthreads();
        if (!s_frozen)
            for (int v = t; v < p.n; v += nt)                         // a6: projected step in shared memory
                if (!p.fixed[v]) {
                    T nx = fma_(-p.eta, sg[v], sx[v]);
                    nx = nx > T(1) ? T(1) : nx;
                    nx = nx < T(-1) ? T(-1) : nx;
                    sx[v] = nx;
                }
    }
    if (t == 0) p.sat_count[b] = last;
    __syncthreads();
    for (int v = t; v < p.n; v += nt) p.x[(int64_t)v * p.ldb + b] = sx[v];
    if (t == 0 && p.h_any) {                                          // the last CTA settles the host copy of the first step
        __threadfence();
        if (atomicAdd(p.d_any + 2, 1) == (int)gridDim.x - 1 && p.d_any[0]) {
            p.h_any[1] = atomicMin(p.d_any + 1, 0x7fffffff);
            __threadfence_system();
            p.h_any[0] = 1;
        }
    }
}

// ---- FP-pipe peak probes (afsat_probe_peak): independent FMA chains, nothing else ----------------------------------
// kind 0: scalar FFMA, 1: packed FFMA2 (fma.rn.f32x2), 2: DFMA.  Every thread runs 8 independent chains.
template <int KIND>
__global__ void __launch_bounds__(256) k_probe(float *out, int iters, float seed)
{
    if (KIND == 0) {
        float a[8], m = seed, c = 0.5f;
#pragma unroll
        for (int j = 0; j < 8; ++j) a[j] = seed + j;
        for (int i = 0; i < iters; ++i)
#pragma unroll
            for (int j = 0; j < 8; ++j) a[j] = fmaf(a[j], m, c);
        float s = 0.f;
#pragma unroll
        for (int j = 0; j < 8; ++j) s += a[j];
        if (s == 12345.678f) out[0] = s;
    } else if (KIND == 1) {
        f32x2 a[8];
        const f32x2 m = pk(seed, seed), c = pk(0.5f, 0.25f);
#pragma unroll
        for (int j = 0; j < 8; ++j) a[j] = pk(seed + j, seed - j);
        for (int i = 0; i < iters; ++i)
#pragma unroll
            for (int j = 0; j < 8; ++j) a[j] = fma2(a[j], m, c);
        f32x2 s = 0ull;
#pragma unroll
        for (int j = 0; j < 8; ++j) s = add2(s, a[j]);
        if (s == 0x123456789ull) out[0] = 1.f;
    } else {
        double a[8], m = seed, c = 0.5;
#pragma unroll
        for (int j = 0; j < 8; ++j) a[j] = seed + j;
        for (int i = 0; i < iters; ++i)
#pragma unroll
            for (int j = 0; j < 8; ++j) a[j] = fma(a[j], m, c);
        double s = 0.;
#pragma unroll
        for (int j = 0; j < 8; ++j) s += a[j];
        if (s == 12345.678) out[0] = (float)s;
    }
}

// kinds 3 / 4 / 5: L2 delivery rate -- every thread walks an L2-resident buffer with 16-byte loads that bypass L1
// (ld.global.cg), 16-byte vector REDs (red.global.add.v4.f32), or both in turn on two halves of the buffer: the access
// kinds of the evaluation kernels (a1 gathers, a5 scatter-adds; they move the same number of bytes each way)
template <int MODE>
__global__ void __launch_bounds__(256) k_probe_l2(float4 *buf, size_t n_vec, int iters, float *out)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x, i0 = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const size_t half = n_vec / 2;
    float acc = 0.f;
    for (int it = 0; it < iters; ++it)
        for (size_t i = i0; i < (MODE == 2 ? half : n_vec); i += stride) {
            if (MODE == 1 || MODE == 2)
                asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(buf + i), "f"(1.0f), "f"(0.5f), "f"(0.25f), "f"(2.0f) : "memory");
            if (MODE == 0 || MODE == 2) {
                float4 v;
                asm volatile("ld.global.cg.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w)
                             : "l"(buf + (MODE == 2 ? half : 0) + i) : "memory");
                acc += v.x + v.y + v.z + v.w;
            }
        }
    if (acc == 12345.678f) out[0] = acc;
}

}  // namespace afsat
