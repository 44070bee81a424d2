// afsat_split.cuh -- lane-split register kernel for LONG fp32 constraints (k > AFSAT_B_KMAX32;
// DESIGN.md 6.2b).  Internal to the library.
//
// One (constraint, candidate) evaluation is shared by NS lanes of a warp: lane (h, c) -- h = lane / (32 / NS),
// c = lane % (32 / NS) -- owns the literals j = i NS + h, i < KS = ceil(k / NS), of candidate c.  Per DFT point
// every lane walks ITS literals forward (prefixes of its own partial product), the NS partial
// products are exchanged with warp shuffles, and the backward walk is seeded with  w b x (product of the OTHER
// lanes' partial products):  the leave-one-out product of literal i in lane h is
//     prefix_h(i) x suffix_h(i) x prod_{h' != h} P_h',
// still a product of factors, never a division (north_star).  Every intermediate of a point -- the KS literal values,
// factors, prefixes and partial gradients of the lane -- then fits in registers WITHOUT spills at k = 64, at twice the
// warps per SM of the one-lane-per-candidate kernel (k_eval_km: 255 registers, spills beyond k ~ 36); the arithmetic
// per literal and point is the same 12 instructions, plus one exchange (2 (NS - 1) shuffles, NS - 1 + 2 complex
// multiplies) per point.  Literals missing from the last row (j >= k) are unit factors.
#pragma once
#include "afsat_internal.h"
#include "afsat_kernels.cuh"

namespace afsat {

#ifndef AFSAT_L32_NS
#define AFSAT_L32_NS 2                 // lanes per (constraint, candidate)
#endif
#ifndef AFSAT_L32_THREADS
#define AFSAT_L32_THREADS 384             // 12 warps per SM at 168 registers (measured: 256 / 255 regs 5 % slower)
#endif
#ifndef AFSAT_L32_MINB
#define AFSAT_L32_MINB 1
#endif
#ifndef AFSAT_L32_CHAINS
#define AFSAT_L32_CHAINS 2             // independent product chains per thread at a complex point
#endif
#ifndef AFSAT_M32_THREADS
#define AFSAT_M32_THREADS 384
#endif
#ifndef AFSAT_L64_THREADS
#define AFSAT_L64_THREADS 384             // 168 registers, 12 warps per SM (256 x 255 registers: 4.25 vs 4.07 ms on cfg3)
#endif
#define AFSAT_L64_KMIN (AFSAT_B_KMAX + 1)   // fp64, k > 20: FOUR lanes per candidate (a double takes two registers)
#ifndef AFSAT_L32_PREFETCH
#define AFSAT_L32_PREFETCH 1
#endif
#ifndef AFSAT_L32_KMIN
#define AFSAT_L32_KMIN (AFSAT_B_KMAX + 1)
#endif

// product of the OTHER lanes' values (NS = 2: the partner's; NS = 4: butterfly over lane bits log2(CW), log2(CW) + 1)
template <typename T, int NS>
__device__ __forceinline__ T others_real(unsigned mask, T v)
{
    constexpr int CW = 32 / NS;
    if (NS == 2) return __shfl_xor_sync(mask, v, CW);
    const T n1 = __shfl_xor_sync(mask, v, CW);
    const T po = __shfl_xor_sync(mask, v * n1, 2 * CW);
    return n1 * po;
}
template <typename T, int NS>
__device__ __forceinline__ void others_cplx(unsigned mask, T vr, T vi, T &orr, T &oi)
{
    constexpr int CW = 32 / NS;
    const T n1r = __shfl_xor_sync(mask, vr, CW), n1i = __shfl_xor_sync(mask, vi, CW);
    if (NS == 2) { orr = n1r; oi = n1i; return; }
    const T ppr = fma_(vr, n1r, -(vi * n1i)), ppi = fma_(vr, n1i, vi * n1r);
    const T por = __shfl_xor_sync(mask, ppr, 2 * CW), poi = __shfl_xor_sync(mask, ppi, 2 * CW);
    orr = fma_(n1r, por, -(n1i * poi)); oi = fma_(n1r, poi, n1i * por);
}

// a2-a4 for the lane's KS literals of one constraint; tab rows as in eval_points_reg ({Re a, Im a, Re b, Im b,
// Re w, Im w, Re(w b), Im(w b)}, real rows first).  miss: the lane's LAST literal does not exist (unit factor).
template <typename T, int KS, int NS, bool GRAD>
__device__ __forceinline__ void eval_points_split(unsigned mask, const T (&y)[KS], bool miss,
                                                  const T *__restrict__ tab, int n_real, int n_cplx, T &fe,
                                                  T (&g)[KS])
{
    const T *r = tab;
    for (int p = 0; p < n_real; ++p, r += 8) {                       // self-conjugate points
        const T a = r[0], b = r[2], w = r[4], wb = r[6];
        T pre[KS], f[KS];
#pragma unroll
        for (int i = 0; i < KS; ++i) f[i] = fma_(b, y[i], a);
        if (miss) f[KS - 1] = T(1);
        T run = f[0];
#pragma unroll
        for (int i = 1; i < KS; ++i) { pre[i] = run; run *= f[i]; }
        const T oth = others_real<T, NS>(mask, run);
        fe = fma_(w, run * oth, fe);
        if (GRAD) {
            T suf = wb * oth;
#pragma unroll
            for (int i = KS - 1; i >= 1; --i) { g[i] = fma_(pre[i], suf, g[i]); suf *= f[i]; }
            g[0] += suf;                                              // prefix_0 = 1
        }
    }
    // complex points: the lane's literals are walked as TWO independent chains, A = [0, KA) and B = [KA, KS) -- the
    // same leave-one-out identity one level down (LOO_i = prefix_A(i) suffix_A(i) P_B others) -- so that a thread
    // always has two dependent FMUL -> FFMA sequences in flight (with 3 warps per scheduler one chain per thread
    // leaves the issue slots idle on fixed-latency waits: profiles/r1_eval_split_cfg3.md)
    constexpr int KA = AFSAT_L32_CHAINS == 2 ? KS / 2 : KS, KB = KS - KA;
    for (int p = 0; p < n_cplx; ++p, r += 8) {                       // one of each conjugate pair
        const T ar = r[0], ai = r[1], br = r[2], bi = r[3], wr = r[4], wi = r[5], wbr = r[6], wbi = r[7];
        T pr[KS], pi[KS], fr[KS], fi[KS];
#pragma unroll
        for (int i = 0; i < KS; ++i) { fr[i] = fma_(br, y[i], ar); fi[i] = fma_(bi, y[i], ai); }
        if (miss) { fr[KS - 1] = T(1); fi[KS - 1] = T(0); }
        T rr = fr[0], ri = fi[0], qr = T(1), qi = T(0);
        if (KB > 0) { qr = fr[KA]; qi = fi[KA]; }
#pragma unroll
        for (int i = 1; i < (KA > KB ? KA : KB); ++i) {
            if (i < KA) {
                pr[i] = rr; pi[i] = ri;
                const T nr = fma_(rr, fr[i], -(ri * fi[i]));
                const T ni = fma_(rr, fi[i], ri * fr[i]);
                rr = nr; ri = ni;
            }
            if (i < KB) {
                pr[KA + i] = qr; pi[KA + i] = qi;
                const T nr = fma_(qr, fr[KA + i], -(qi * fi[KA + i]));
                const T ni = fma_(qr, fi[KA + i], qi * fr[KA + i]);
                qr = nr; qi = ni;
            }
        }
        T lr = rr, li = ri;                                       // the lane's partial product P_A P_B
        if (KB > 0) { lr = fma_(rr, qr, -(ri * qi)); li = fma_(rr, qi, ri * qr); }
        T orr, oi;
        others_cplx<T, NS>(mask, lr, li, orr, oi);
        const T tr = fma_(lr, orr, -(li * oi)), ti = fma_(lr, oi, li * orr);   // P_l, the whole product
        fe = fma_(wr, tr, fe);
        fe = fma_(-wi, ti, fe);
        if (GRAD) {
            const T zr = fma_(wbr, orr, -(wbi * oi)), zi = fma_(wbr, oi, wbi * orr);   // w b x others
            T sr = zr, si = zi, ur = zr, ui = zi;                 // suffix of chain A seeded with z P_B, of B with z P_A
            if (KB > 0) {
                sr = fma_(zr, qr, -(zi * qi)); si = fma_(zr, qi, zi * qr);
                ur = fma_(zr, rr, -(zi * ri)); ui = fma_(zr, ri, zi * rr);
            }
#pragma unroll
            for (int i = (KA > KB ? KA : KB) - 1; i >= 1; --i) {
                if (i < KA) {
                    g[i] = fma_(pr[i], sr, g[i]);
                    g[i] = fma_(-pi[i], si, g[i]);
                    const T nr = fma_(sr, fr[i], -(si * fi[i]));
                    const T ni = fma_(sr, fi[i], si * fr[i]);
                    sr = nr; si = ni;
                }
                if (i < KB) {
                    g[KA + i] = fma_(pr[KA + i], ur, g[KA + i]);
                    g[KA + i] = fma_(-pi[KA + i], ui, g[KA + i]);
                    const T nr = fma_(ur, fr[KA + i], -(ui * fi[KA + i]));
                    const T ni = fma_(ur, fi[KA + i], ui * fr[KA + i]);
                    ur = nr; ui = ni;
                }
            }
            g[0] += sr;                                               // prefix_0 = 1 in both chains
            if (KB > 0) g[KA] += ur;
        }
    }
}

template <typename T, int KS, int NS, bool GRAD>
__device__ __forceinline__ void run_item_split(const EvalParams<T> &p, unsigned mask, const int32_t *__restrict__ s_lits,
                                               const T *__restrict__ s_tab, int n_real, int n_cplx, int nc, int wk,
                                               int h, int64_t b, T &fe, int k)
{
    const char *xb = reinterpret_cast<const char *>(p.x + b);
    char *gb = reinterpret_cast<char *>(p.G + (b - p.g_b0));
    const uint32_t x_ld = (uint32_t)(p.ldb * (int64_t)sizeof(T)), g_ld = (uint32_t)(p.g_ld * (int64_t)sizeof(T));
    const int Wk = p.Wk;
    const bool miss = (KS - 1) * NS + h >= k;
    for (int c = wk; c < nc; c += Wk) {
        const int32_t *L = s_lits + c * k + h;
        int32_t lit[KS];
        T y[KS], g[KS];
#pragma unroll
        for (int i = 0; i < KS - 1; ++i) lit[i] = L[i * NS];
        lit[KS - 1] = miss ? LIT_NONE : L[(KS - 1) * NS];             // missing literal: constant, no gather, no RED
#pragma unroll
        for (int i = 0; i < KS; ++i) {
            if (i == KS - 1 && (lit[i] & LIT_NONE)) y[i] = T(1);
            else y[i] = __ldg(reinterpret_cast<const T *>(xb + (uint64_t)(uint32_t)(lit[i] & LIT_VAR) * x_ld));
            y[i] = flip_sign(y[i], lit[i]);
            g[i] = T(0);
        }
#if AFSAT_L32_PREFETCH
        if (c + Wk < nc) {                                            // the NEXT constraint's row segments into L1: with 2-3
            const int32_t *Ln = L + Wk * k;                           // warps per scheduler nothing else hides its gathers
#pragma unroll
            for (int i = 0; i < KS; ++i) {
                if (i == KS - 1 && miss) continue;
                const int32_t ln = Ln[i * NS];
                asm volatile("prefetch.global.L1 [%0];" ::"l"(xb + (uint64_t)(uint32_t)(ln & LIT_VAR) * x_ld));
            }
        }
#endif
        eval_points_split<T, KS, NS, GRAD>(mask, y, miss, s_tab, n_real, n_cplx, fe, g);
        if (GRAD) {
#pragma unroll
            for (int i = 0; i < KS; ++i) {
                if (i == KS - 1 && (lit[i] & LIT_NONE)) continue;
                const T gi[1] = {flip_sign(g[i], lit[i])};
                VecIO<T, 1>::red(reinterpret_cast<T *>(gb + (uint64_t)(uint32_t)(lit[i] & LIT_VAR) * g_ld), gi);
            }
        }
    }
}

template <typename T, int KS, int NS, bool GRAD>
__device__ __noinline__ void item_body_split(const EvalParams<T> &p, const int32_t *s_lits, const T *s_tab,
                                             T (*s_F)[32], int n_real, int n_cplx, int nc, int k)
{
    constexpr int CW = 32 / NS;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int h = lane / CW, cl = lane % CW;
    const int wc = warp % p.Wc, wk = warp / p.Wc;
    const int64_t b = p.b_begin + ((int64_t)blockIdx.y * p.Wc + wc) * CW + cl;
    const bool active = b < p.b_end && b < p.B && !lane_skipped(p, b, 1);   // the NS lanes of a candidate agree
    const unsigned mask = __ballot_sync(0xffffffffu, active);
    T fe = T(0);
    if (active) {
        run_item_split<T, KS, NS, GRAD>(p, mask, s_lits, s_tab, n_real, n_cplx, nc, wk, h, b, fe, k);
    }
    if (!p.Fpart) return;
    s_F[warp][lane] = fe;
    __syncthreads();
    if (wk == 0 && h == 0 && active) {                                // fixed order over the Wk constraint groups
        T s = T(0);
        for (int g = 0; g < p.Wk; ++g) s += s_F[warp + g * p.Wc][lane];
        p.Fpart[(int64_t)(p.frow_base + blockIdx.x) * p.ldb + b] = s;
    }
}

// ---- packed form (V = 2): a lane holds TWO adjacent candidates as f32x2 pairs and every product is an FFMA2 / FMUL2
// (DESIGN.md 6.1 "FFMA2"): half the issue slots for the same flops.  FFMA2 has no negated operands, so -Im f is made by
// XOR on the ALU pipe and the backward walk carries the suffix as (Re s, -Im s).  12 registers per literal, so this
// form serves the lengths whose KS fits the register budget (9 <= k <= AFSAT_B_KMAX32).
constexpr f32x2 SGN2 = 0x8000000080000000ull;
__device__ __forceinline__ f32x2 shfl2(unsigned mask, f32x2 v, int d)
{
    float lo, hi; upk(v, lo, hi);
    return pk(__shfl_xor_sync(mask, lo, d), __shfl_xor_sync(mask, hi, d));
}

template <int KS, int NS, bool GRAD>
__device__ __forceinline__ void eval_points_split2(unsigned mask, const f32x2 (&y)[KS], bool miss,
                                                   const float *__restrict__ tab, int n_real, int n_cplx, f32x2 &fe,
                                                   f32x2 (&g)[KS])
{
    static_assert(NS == 2, "the packed form exchanges with one partner");
    constexpr int CW = 32 / NS;
    const f32x2 one2 = pk(1.0f, 1.0f);
    const float *r = tab;
    for (int p = 0; p < n_real; ++p, r += 8) {                       // self-conjugate points
        const f32x2 a = pk(r[0], r[0]), b = pk(r[2], r[2]), w = pk(r[4], r[4]), wb = pk(r[6], r[6]);
        f32x2 pre[KS], f[KS];
#pragma unroll
        for (int i = 0; i < KS; ++i) f[i] = fma2(b, y[i], a);
        if (miss) f[KS - 1] = one2;
        f32x2 run = f[0];
#pragma unroll
        for (int i = 1; i < KS; ++i) { pre[i] = run; run = mul2(run, f[i]); }
        const f32x2 oth = shfl2(mask, run, CW);
        fe = fma2(w, mul2(run, oth), fe);
        if (GRAD) {
            f32x2 suf = mul2(wb, oth);
#pragma unroll
            for (int i = KS - 1; i >= 1; --i) { g[i] = fma2(pre[i], suf, g[i]); suf = mul2(suf, f[i]); }
            g[0] = add2(g[0], suf);                                   // prefix_0 = 1
        }
    }
    for (int p = 0; p < n_cplx; ++p, r += 8) {                       // one of each conjugate pair
        const f32x2 ar = pk(r[0], r[0]), ai = pk(r[1], r[1]), br = pk(r[2], r[2]), bi = pk(r[3], r[3]);
        f32x2 pr[KS], pi[KS], fr[KS], fi[KS];
#pragma unroll
        for (int i = 0; i < KS; ++i) { fr[i] = fma2(br, y[i], ar); fi[i] = fma2(bi, y[i], ai); }
        if (miss) { fr[KS - 1] = one2; fi[KS - 1] = 0ull; }
        f32x2 rr = fr[0], ri = fi[0];
#pragma unroll
        for (int i = 1; i < KS; ++i) {
            pr[i] = rr; pi[i] = ri;
            const f32x2 nr = fma2(rr, fr[i], mul2(ri, fi[i] ^ SGN2));   // Re: rr fr - ri fi
            const f32x2 ni = fma2(rr, fi[i], mul2(ri, fr[i]));          // Im: rr fi + ri fr
            rr = nr; ri = ni;
        }
        const f32x2 orr = shfl2(mask, rr, CW), oi = shfl2(mask, ri, CW);
        const f32x2 tr = fma2(rr, orr, mul2(ri, oi ^ SGN2)), ti = fma2(rr, oi, mul2(ri, orr));   // P_l, the whole product
        fe = fma2(pk(r[4], r[4]), tr, fe);
        fe = fma2(pk(-r[5], -r[5]), ti, fe);
        if (GRAD) {
            const f32x2 wbr = pk(r[6], r[6]), wbi = pk(r[7], r[7]);
            f32x2 sr = fma2(wbr, orr, mul2(wbi, oi ^ SGN2));           // suffix (Re s, -Im s) seeded with w b x other
            f32x2 nsi = fma2(wbr, oi, mul2(wbi, orr)) ^ SGN2;
#pragma unroll
            for (int i = KS - 1; i >= 1; --i) {
                g[i] = fma2(pr[i], sr, g[i]);
                g[i] = fma2(pi[i], nsi, g[i]);                        // Re(prefix x suffix)
                const f32x2 nr = fma2(sr, fr[i], mul2(nsi, fi[i]));
                const f32x2 nn = fma2(nsi, fr[i], mul2(sr, fi[i] ^ SGN2));
                sr = nr; nsi = nn;
            }
            g[0] = add2(g[0], sr);                                    // prefix_0 = 1
        }
    }
}

template <int KS, int NS, bool GRAD>
__device__ __forceinline__ void run_item_split2(const EvalParams<float> &p, unsigned mask, const int32_t *__restrict__ s_lits,
                                                const float *__restrict__ s_tab, int n_real, int n_cplx, int nc, int wk,
                                                int h, int64_t b, f32x2 &fe, int k)
{
    const char *xb = reinterpret_cast<const char *>(p.x + b);
    char *gb = reinterpret_cast<char *>(p.G + (b - p.g_b0));
    const uint32_t x_ld = (uint32_t)(p.ldb * 4), g_ld = (uint32_t)(p.g_ld * 4);
    const int Wk = p.Wk;
    const bool miss = (KS - 1) * NS + h >= k;
    const f32x2 one2 = pk(1.0f, 1.0f);
    for (int c = wk; c < nc; c += Wk) {
        const int32_t *L = s_lits + c * k + h;
        int32_t lit[KS];
        f32x2 y[KS], g[KS];
#pragma unroll
        for (int i = 0; i < KS - 1; ++i) lit[i] = L[i * NS];
        lit[KS - 1] = miss ? LIT_NONE : L[(KS - 1) * NS];             // missing literal: constant, no gather, no RED
#pragma unroll
        for (int i = 0; i < KS; ++i) {
            f32x2 v[1] = {one2};
            if (!(i == KS - 1 && (lit[i] & LIT_NONE)))
                PairIO<1>::load(xb + (uint64_t)(uint32_t)(lit[i] & LIT_VAR) * x_ld, v);
            const uint32_t m = (uint32_t)(lit[i] & LIT_NEG);
            y[i] = v[0] ^ (((f32x2)m << 32) | m);                     // y = s x
            g[i] = 0ull;
        }
#if AFSAT_L32_PREFETCH
        if (c + Wk < nc) {
            const int32_t *Ln = L + Wk * k;
#pragma unroll
            for (int i = 0; i < KS; ++i) {
                if (i == KS - 1 && miss) continue;
                const int32_t ln = Ln[i * NS];
                asm volatile("prefetch.global.L1 [%0];" ::"l"(xb + (uint64_t)(uint32_t)(ln & LIT_VAR) * x_ld));
            }
        }
#endif
        eval_points_split2<KS, NS, GRAD>(mask, y, miss, s_tab, n_real, n_cplx, fe, g);
        if (GRAD) {
#pragma unroll
            for (int i = 0; i < KS; ++i) {
                if (i == KS - 1 && (lit[i] & LIT_NONE)) continue;
                const uint32_t m = (uint32_t)(lit[i] & LIT_NEG);
                const f32x2 gi[1] = {g[i] ^ (((f32x2)m << 32) | m)};
                PairIO<1>::red(gb + (uint64_t)(uint32_t)(lit[i] & LIT_VAR) * g_ld, gi);
            }
        }
    }
}

template <int KS, int NS, bool GRAD>
__device__ __noinline__ void item_body_split2(const EvalParams<float> &p, const int32_t *s_lits, const float *s_tab,
                                              float (*s_F)[64], int n_real, int n_cplx, int nc, int k)
{
    constexpr int CW = 32 / NS;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int h = lane / CW, cl = lane % CW;
    const int wc = warp % p.Wc, wk = warp / p.Wc;
    const int64_t b = p.b_begin + ((int64_t)blockIdx.y * p.Wc + wc) * (2 * CW) + 2 * cl;
    const bool active = b < p.b_end && b < p.B && !lane_skipped(p, b, 2);   // the NS lanes of a candidate pair agree
    const unsigned mask = __ballot_sync(0xffffffffu, active);
    f32x2 fe2 = 0ull;
    if (active) {
        run_item_split2<KS, NS, GRAD>(p, mask, s_lits, s_tab, n_real, n_cplx, nc, wk, h, b, fe2, k);
    }
    if (!p.Fpart) return;
    float f0, f1; upk(fe2, f0, f1);
    s_F[warp][2 * lane] = f0; s_F[warp][2 * lane + 1] = f1;
    __syncthreads();
    if (wk == 0 && h == 0 && active) {                                // fixed order over the Wk constraint groups
#pragma unroll
        for (int v = 0; v < 2; ++v) {
            float s = 0.0f;
            for (int g = 0; g < p.Wk; ++g) s += s_F[warp + g * p.Wc][2 * lane + v];
            if (b + v < p.B) p.Fpart[(int64_t)(p.frow_base + blockIdx.x) * p.ldb + b + v] = s;
        }
    }
}

template <typename T, int KS, int KSHI, int NS, int V, bool GRAD>
struct SwitchSplit {
    static __device__ __forceinline__ void go(int ks, const EvalParams<T> &p, const int32_t *s_lits, const T *s_tab,
                                              T (*s_F)[32 * V], int n_real, int n_cplx, int nc, int k)
    {
        if (ks == KS) {
            if constexpr (V == 2) item_body_split2<KS, NS, GRAD>(p, s_lits, s_tab, s_F, n_real, n_cplx, nc, k);
            else item_body_split<T, KS, NS, GRAD>(p, s_lits, s_tab, s_F, n_real, n_cplx, nc, k);
        } else if (KS < KSHI)
            SwitchSplit<T, (KS < KSHI ? KS + 1 : KS), KSHI, NS, V, GRAD>::go(ks, p, s_lits, s_tab, s_F, n_real, n_cplx, nc, k);
    }
};

// one launch for every length in [KLO, KHI]: the CTA's item picks the body compiled for ceil(k / NS) literals per lane
template <typename T, int KLO, int KHI, int NS, int V, bool GRAD, int THREADS, int MINB>
__global__ void __launch_bounds__(THREADS, MINB) k_eval_split(const EvalParams<T> p)
{
    __shared__ __align__(16) T s_tab[((KHI + 1) / 2 + 1) * 8];
    __shared__ int32_t s_lits[LIT_CHUNK];
    __shared__ T s_F[THREADS / 32][32 * V];
    const Item it = p.items[blockIdx.x];
    const SigDev sg = p.sigs[it.sig];
    stage_item(p, it, sg, s_tab, s_lits);
    __syncthreads();
    SwitchSplit<T, (KLO + NS - 1) / NS, (KHI + NS - 1) / NS, NS, V, GRAD>::go((it.k + NS - 1) / NS, p, s_lits, s_tab, s_F, sg.n_real,
                                                                        sg.n_cplx, it.c_end - it.c_begin, it.k);
}

#ifndef AFSAT_KS32_TU   // instantiated in afsat_ks32.cu
extern template __global__ void k_eval_split<float, AFSAT_L32_KMIN, AFSAT_MAX_LEN, AFSAT_L32_NS, 1, true, AFSAT_L32_THREADS, AFSAT_L32_MINB>(const EvalParams<float>);
extern template __global__ void k_eval_split<float, AFSAT_L32_KMIN, AFSAT_MAX_LEN, AFSAT_L32_NS, 1, false, AFSAT_L32_THREADS, AFSAT_L32_MINB>(const EvalParams<float>);
extern template __global__ void k_eval_split<double, AFSAT_L64_KMIN, AFSAT_MAX_LEN, 4, 1, true, AFSAT_L64_THREADS, 1>(const EvalParams<double>);
extern template __global__ void k_eval_split<double, AFSAT_L64_KMIN, AFSAT_MAX_LEN, 4, 1, false, AFSAT_L64_THREADS, 1>(const EvalParams<double>);
extern template __global__ void k_eval_split<float, AFSAT_A_KMAX + 1, AFSAT_B_KMAX, 2, 2, true, AFSAT_M32_THREADS, 1>(const EvalParams<float>);
extern template __global__ void k_eval_split<float, AFSAT_A_KMAX + 1, AFSAT_B_KMAX, 2, 2, false, AFSAT_M32_THREADS, 1>(const EvalParams<float>);
#endif

}  // namespace afsat
