// afsat_split.cuh -- lane-split register kernels for constraints too long for one lane per candidate (SURVEY.md §8(a)
// a1-a5: fp32 k > 8, fp64 k > 20).  Internal to the library.
//
// One (constraint, candidate) evaluation is shared by NS lanes of a warp: lane (h, c) -- h = lane / (32 / NS),
// c = lane % (32 / NS) -- owns the literals j = i NS + h, i < KS = ceil(k / NS), of candidate c.  Per DFT point
// every lane forms the partial product of ITS literals, the NS partial products are exchanged with warp
// shuffles, and the backward walk is seeded with  w x (product of the OTHER lanes' partial products): a leave-one-out
// product is always prefix x suffix x the others' products, still a product of factors, never a division (north_star).
//
// Literal GROUPS (scalar form).  Inside a lane the literals are taken M at a time: the product of a group's factors is
// the polynomial  prod_{u<M} (a + b y_u) = sum_{j<=M} a^(M-j) b^j e_j(y_group)  in its M + 1 elementary symmetric
// polynomials, which do not depend on the DFT point -- they are formed once per constraint -- so at every point a group
// costs 2 M FMAs for its (complex) factor instead of M factors and M - 1 complex multiplies, the prefix / suffix walk
// runs over ceil(KS / M) group factors instead of KS, and the partial gradients come out of M accumulators per group,
//     A_j += Re( w a^(M-j) b^j x prefix_g x suffix_g x others ),     dFE/dy_u = sum_j A_j e_{j-1}(y_group without y_u),
// expanded once per constraint.  Per literal and complex point that is 4 + 12 / M instructions instead of 12 (M = 4: 7);
// the generating polynomial is still evaluated at every DFT point and contracted with the same weights -- the groups
// only change the order in which its factors are multiplied.  A slot without a literal (k not a multiple of NS, KS not
// a multiple of M) holds the value `pad` for which the factor is exactly 1 at every point: 0 for the paper's tables
// (staged un-halved, a = 1, b = w^l, the 2^-k folded into the weights -- an exact rescale), 1 for the robust tables
// (a + b = 1).
#pragma once
#include "afsat_internal.h"
#include "afsat_kernels.cuh"

namespace afsat {

#define AFSAT_L32_NS 2                 // lanes per (constraint, candidate)
#define AFSAT_L32_THREADS 384             // 12 warps per SM at 168 registers (cfg3, ms / step: 256: 1.66, 320: 1.72, 384: 1.53, 512: 1.57)
#define AFSAT_L32_MINB 1
#define AFSAT_M32_THREADS 256             // packed form, k <= 20: 2 CTAs x 8 warps at 128 registers (cfg2: 0.621 ms / step against
                                          // 0.651 with 384 threads x 168 registers and 0.637 with 512 x 128)
#define AFSAT_M32_MINB 2
#define AFSAT_L64_THREADS 384
#define AFSAT_L64_KMIN (AFSAT_B_KMAX + 1)   // fp64, k > 20: FOUR lanes per candidate (a double takes two registers)
#define AFSAT_L32_KMIN (AFSAT_B_KMAX + 1)
// Group layout of a lane with KS literal slots: NG = ceil(KS / 4) groups of BALANCED sizes -- the first NHI = KS mod NG
// groups take MHI = MLO + 1 literals, the others MLO = floor(KS / NG) (<= 4) -- so that no slot is wasted on padding.
// Staged row of a point: {Re, Im of c_0 .. c_MHI for groups of MHI | the same for groups of MLO (from scalar ROWG_LO) |
// Re w, Im w (at ROWG_W)},  c_j = a^(M-j) b^j.
constexpr int GRP_MAX = 4;
constexpr int ROWG_LO = 2 * (GRP_MAX + 1), ROWG_W = 4 * (GRP_MAX + 1), ROWG = ROWG_W + 4;   // 24: rows are whole 16-byte vectors
struct GrpLayout { int NG, MLO, NHI, MHI; };
__host__ __device__ constexpr GrpLayout grp_layout(int KS)
{
    const int NG = (KS + GRP_MAX - 1) / GRP_MAX, MLO = KS / NG, NHI = KS % NG;
    return GrpLayout{NG, MLO, NHI, MLO + (NHI > 0 ? 1 : 0)};
}
__host__ __device__ constexpr int grp_size(const GrpLayout &L, int gq) { return gq < L.NHI ? L.MHI : L.MLO; }
__host__ __device__ constexpr int grp_off(const GrpLayout &L, int gq) { return gq < L.NHI ? gq * L.MHI : L.NHI * L.MHI + (gq - L.NHI) * L.MLO; }

// HOST: the staged table of one signature for the grouped kernels, from its rows {Re a, Im a, Re b, Im b, Re w, Im w, ..}
// (real rows first), for lanes of KS = ceil(k / NS) slots.  The paper's tables (a = 1/2 in every row) are staged
// un-halved (see above).  Returns the pad value (0 or 1).
inline int pack_rows_grp(const double *r0, int n_rows, int k, int ns, double *out)
{
    bool std_tab = true;
    for (int q = 0; q < n_rows; ++q) std_tab = std_tab && r0[8 * q] == 0.5 && r0[8 * q + 1] == 0.0;
    const double sc = std_tab ? 2.0 : 1.0;
    double scw = 1.0;
    if (std_tab) for (int i = 0; i < k; ++i) scw *= 0.5;
    const GrpLayout L = grp_layout((k + ns - 1) / ns);
    const int M[2] = {L.MHI, L.MLO}, off[2] = {0, ROWG_LO};
    for (int q = 0; q < n_rows; ++q) {
        const double *r = r0 + 8 * q;
        double *o = out + (size_t)q * ROWG;
        for (int j = 0; j < ROWG; ++j) o[j] = 0.0;
        const double ar = sc * r[0], ai = sc * r[1], br = sc * r[2], bi = sc * r[3];
        // a^(M-j) b^j by repeated multiplication of double-precision values (M <= 4: relative error ~1e-15)
        for (int gq = 0; gq < 2; ++gq)
            for (int j = 0; j <= M[gq]; ++j) {
                double cr = 1.0, ci = 0.0;
                for (int t = 0; t < M[gq]; ++t) {
                    const double fr = t < j ? br : ar, fi = t < j ? bi : ai;
                    const double nr = cr * fr - ci * fi, ni = cr * fi + ci * fr;
                    cr = nr; ci = ni;
                }
                o[off[gq] + 2 * j] = cr; o[off[gq] + 2 * j + 1] = ci;
            }
        o[ROWG_W] = r[4] * scw; o[ROWG_W + 1] = r[5] * scw;
    }
    return std_tab ? 0 : 1;
}

// one staged row into registers with 16-byte shared-memory loads (the row is warp-uniform: broadcast)
__device__ __forceinline__ void load_row(const float *__restrict__ r, float (&v)[ROWG])
{
    const float4 *r4 = reinterpret_cast<const float4 *>(r);
#pragma unroll
    for (int i = 0; i < ROWG / 4; ++i) { const float4 t = r4[i]; v[4 * i] = t.x; v[4 * i + 1] = t.y; v[4 * i + 2] = t.z; v[4 * i + 3] = t.w; }
}
__device__ __forceinline__ void load_row(const double *__restrict__ r, double (&v)[ROWG])
{
    const double2 *r2 = reinterpret_cast<const double2 *>(r);
#pragma unroll
    for (int i = 0; i < ROWG / 2; ++i) { const double2 t = r2[i]; v[2 * i] = t.x; v[2 * i + 1] = t.y; }
}

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

// a2-a4 for the lane's KS literal slots of one constraint (a slot without a literal holds the pad value); tab: ROWG scalars
// per retained DFT point, real points first.  Returns the lane's partial gradients dFE/dy_i in g.
template <typename T, int KS, int NS, bool GRAD>
__device__ __forceinline__ void eval_points_grp(unsigned mask, const T (&y)[KS], const T *__restrict__ tab, int n_real,
                                                int n_cplx, T &fe, T (&g)[KS])
{
    constexpr GrpLayout L = grp_layout(KS);
    constexpr int NG = L.NG, MX = L.MHI;
    T e[NG][MX], A[NG][MX];                                          // e[g][j-1] = e_j(group g); A[g][j-1] pairs with c_j
#pragma unroll
    for (int gq = 0; gq < NG; ++gq) {
        const int Mg = grp_size(L, gq), off = grp_off(L, gq);
        T ee[MX + 1];
        ee[0] = T(1);
#pragma unroll
        for (int j = 1; j <= MX; ++j) ee[j] = T(0);
#pragma unroll
        for (int u = 0; u < MX; ++u)
            if (u < Mg) {
                const T yv = y[off + u < KS ? off + u : 0];
#pragma unroll
                for (int j = MX; j >= 1; --j)
                    if (j <= u + 1) ee[j] = fma_(yv, ee[j - 1], ee[j]);
            }
#pragma unroll
        for (int j = 0; j < MX; ++j) { e[gq][j] = ee[j + 1]; A[gq][j] = T(0); }
    }
    const T *r = tab;
    for (int p = 0; p < n_real; ++p, r += ROWG) {                    // self-conjugate points
        T rv[ROWG], ch[MX + 1], cl[MX + 1];
        load_row(r, rv);
#pragma unroll
        for (int j = 0; j <= MX; ++j) { ch[j] = rv[2 * j]; cl[j] = rv[ROWG_LO + 2 * j]; }
        const T w = rv[ROWG_W];
        T q[NG], pre[NG];
#pragma unroll
        for (int gq = 0; gq < NG; ++gq) {
            const int Mg = grp_size(L, gq);
            const bool hi = gq < L.NHI;
            T sacc = hi ? ch[0] : cl[0];
#pragma unroll
            for (int j = 0; j < MX; ++j)
                if (j < Mg) sacc = fma_(hi ? ch[j + 1] : cl[j + 1], e[gq][j], sacc);
            q[gq] = sacc;
        }
        T run = q[0];
#pragma unroll
        for (int gq = 1; gq < NG; ++gq) { pre[gq] = run; run *= q[gq]; }
        const T oth = others_real<T, NS>(mask, run);
        T suf = w * oth;
        fe = fma_(suf, run, fe);
        if (GRAD) {
#pragma unroll
            for (int gq = NG - 1; gq >= 0; --gq) {
                const int Mg = grp_size(L, gq);
                const bool hi = gq < L.NHI;
                const T t = gq > 0 ? pre[gq] * suf : suf;
#pragma unroll
                for (int j = 0; j < MX; ++j)
                    if (j < Mg) A[gq][j] = fma_(hi ? ch[j + 1] : cl[j + 1], t, A[gq][j]);
                if (gq > 0) suf *= q[gq];
            }
        }
    }
    for (int p = 0; p < n_cplx; ++p, r += ROWG) {                    // one of each conjugate pair
        T rv[ROWG], chr[MX + 1], chi[MX + 1], clr[MX + 1], cli[MX + 1];
        load_row(r, rv);
#pragma unroll
        for (int j = 0; j <= MX; ++j) {
            chr[j] = rv[2 * j]; chi[j] = rv[2 * j + 1];
            clr[j] = rv[ROWG_LO + 2 * j]; cli[j] = rv[ROWG_LO + 2 * j + 1];
        }
        const T wr = rv[ROWG_W], wi = rv[ROWG_W + 1];
        T qr[NG], qi[NG], pr[NG], pi[NG];
#pragma unroll
        for (int gq = 0; gq < NG; ++gq) {
            const int Mg = grp_size(L, gq);
            const bool hi = gq < L.NHI;
            T sr = hi ? chr[0] : clr[0], si = hi ? chi[0] : cli[0];
#pragma unroll
            for (int j = 0; j < MX; ++j)
                if (j < Mg) { sr = fma_(hi ? chr[j + 1] : clr[j + 1], e[gq][j], sr); si = fma_(hi ? chi[j + 1] : cli[j + 1], e[gq][j], si); }
            qr[gq] = sr; qi[gq] = si;
        }
        T rr = qr[0], ri = qi[0];
#pragma unroll
        for (int gq = 1; gq < NG; ++gq) {
            pr[gq] = rr; pi[gq] = ri;
            const T nr = fma_(rr, qr[gq], -(ri * qi[gq]));
            const T ni = fma_(rr, qi[gq], ri * qr[gq]);
            rr = nr; ri = ni;
        }
        T orr, oi;
        others_cplx<T, NS>(mask, rr, ri, orr, oi);
        T sr = fma_(wr, orr, -(wi * oi)), si = fma_(wr, oi, wi * orr);      // suffix seeded with w x others
        fe = fma_(sr, rr, fe);
        fe = fma_(-si, ri, fe);                                              // Re(w others P_lane)
        if (GRAD) {
#pragma unroll
            for (int gq = NG - 1; gq >= 0; --gq) {
                const int Mg = grp_size(L, gq);
                const bool hi = gq < L.NHI;
                T tr = sr, ti = si;
                if (gq > 0) { tr = fma_(pr[gq], sr, -(pi[gq] * si)); ti = fma_(pr[gq], si, pi[gq] * sr); }
#pragma unroll
                for (int j = 0; j < MX; ++j)
                    if (j < Mg) {
                        A[gq][j] = fma_(hi ? chr[j + 1] : clr[j + 1], tr, A[gq][j]);
                        A[gq][j] = fma_(-(hi ? chi[j + 1] : cli[j + 1]), ti, A[gq][j]);   // Re(c_j T)
                    }
                if (gq > 0) {
                    const T nr = fma_(sr, qr[gq], -(si * qi[gq]));
                    const T ni = fma_(sr, qi[gq], si * qr[gq]);
                    sr = nr; si = ni;
                }
            }
        }
    }
    if (GRAD) {                                                       // dFE/dy_u = sum_j A_j e_{j-1}(group without y_u)
#pragma unroll
        for (int gq = 0; gq < NG; ++gq) {
            const int Mg = grp_size(L, gq), off = grp_off(L, gq);
#pragma unroll
            for (int u = 0; u < MX; ++u) {
                if (u >= Mg) continue;
                T ee[MX];
                ee[0] = T(1);
#pragma unroll
                for (int j = 1; j < MX; ++j) ee[j] = T(0);
                int cntv = 0;
#pragma unroll
                for (int v = 0; v < MX; ++v) {
                    if (v == u || v >= Mg) continue;
                    const T yv = y[off + v < KS ? off + v : 0];
#pragma unroll
                    for (int j = MX - 1; j >= 1; --j)
                        if (j <= cntv + 1) ee[j] = fma_(yv, ee[j - 1], ee[j]);
                    ++cntv;
                }
                T acc = A[gq][0];
#pragma unroll
                for (int j = 1; j < MX; ++j)
                    if (j < Mg) acc = fma_(A[gq][j], ee[j], acc);
                g[off + u < KS ? off + u : 0] = acc;
            }
        }
    }
}

template <typename T, int KS, int NS, bool GRAD>
__device__ __forceinline__ void run_item_split(const EvalParams<T> &p, unsigned mask, const int32_t *__restrict__ s_lits,
                                               const T *__restrict__ s_tab, int n_real, int n_cplx, int nc, int wk,
                                               int h, int64_t b, T &fe, int k, T pad)
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
        lit[KS - 1] = miss ? LIT_NONE : L[(KS - 1) * NS];             // missing literal: the pad value, no gather, no RED
#pragma unroll
        for (int i = 0; i < KS; ++i) {
            if (i == KS - 1 && (lit[i] & LIT_NONE)) y[i] = pad;
            else y[i] = flip_sign(__ldg(reinterpret_cast<const T *>(xb + (uint64_t)(uint32_t)(lit[i] & LIT_VAR) * x_ld)), lit[i]);
            g[i] = T(0);
        }
        if (c + Wk < nc) {                                            // the NEXT constraint's row segments into L1: with 2-3
            const int32_t *Ln = L + Wk * k;                           // warps per scheduler nothing else hides its gathers
#pragma unroll
            for (int i = 0; i < KS; ++i) {
                if (i == KS - 1 && miss) continue;
                const int32_t ln = Ln[i * NS];
                asm volatile("prefetch.global.L1 [%0];" ::"l"(xb + (uint64_t)(uint32_t)(ln & LIT_VAR) * x_ld));
            }
        }
        eval_points_grp<T, KS, NS, GRAD>(mask, y, s_tab, n_real, n_cplx, fe, g);
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
__device__ __forceinline__ void item_body_split(const EvalParams<T> &p, const int32_t *s_lits, const T *s_tab,
                                             T (*s_F)[32], int n_real, int n_cplx, int nc, int k, T pad)
{
    constexpr int CW = 32 / NS;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int h = lane / CW, cl = lane % CW;
    const int wc = warp % p.Wc, wk = warp / p.Wc;
    const int64_t b = p.b_begin + ((int64_t)blockIdx.y * p.Wc + wc) * CW + cl;
    const bool active = b < p.b_end && b < p.B && !lane_skipped(p, b, 1);   // the NS lanes of a candidate agree
    const unsigned mask = __ballot_sync(0xffffffffu, active);
    T fe = T(0);
    if (active) run_item_split<T, KS, NS, GRAD>(p, mask, s_lits, s_tab, n_real, n_cplx, nc, wk, h, b, fe, k, pad);
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
// (DESIGN.md 6.1 "FFMA2"): half the issue slots for the same flops.  The same literal groups as the scalar form, with the
// group coefficients fed through FFMA2's broadcast operand; FFMA2 has no negated operands, so the three negations a
// group needs per point (-Im q, -Im suffix, -Im T) are XORs on the ALU pipe.  Serves 9 <= k <= 20 in fp32.
constexpr f32x2 SGN2 = 0x8000000080000000ull;
__device__ __forceinline__ f32x2 shfl2(unsigned mask, f32x2 v, int d)
{
    float lo, hi; upk(v, lo, hi);
    return pk(__shfl_xor_sync(mask, lo, d), __shfl_xor_sync(mask, hi, d));
}

// group gq of a packed lane: its symmetric polynomials / its share of the gradient, sizes resolved at compile time
template <int KS, int GQ>
__device__ __forceinline__ void grp2_esp(const f32x2 (*y1)[1], f32x2 (*e)[1])
{
    constexpr GrpLayout L = grp_layout(KS);
    constexpr int Mg = grp_size(L, GQ), off = grp_off(L, GQ);
    f32x2 ee[Mg][1];
    esp_f2<Mg, 1>(y1 + off, ee);
#pragma unroll
    for (int j = 0; j < Mg; ++j) e[j][0] = ee[j][0];
}
template <int KS, int GQ>
__device__ __forceinline__ void grp2_loo(const f32x2 (*y1)[1], const f32x2 (*A)[1], f32x2 (*g1)[1])
{
    constexpr GrpLayout L = grp_layout(KS);
    constexpr int Mg = grp_size(L, GQ), off = grp_off(L, GQ);
    f32x2 AA[Mg][1];
#pragma unroll
    for (int j = 0; j < Mg; ++j) AA[j][0] = A[j][0];
    loo_f2<Mg, 1>(y1 + off, AA, g1 + off);
}

template <int KS, int NS, bool GRAD>
__device__ __forceinline__ void eval_points_grp2(unsigned mask, const f32x2 (&y)[KS], const float *__restrict__ tab,
                                                 int n_real, int n_cplx, f32x2 &fe, f32x2 (&g)[KS])
{
    static_assert(NS == 2, "the packed form exchanges with one partner");
    constexpr GrpLayout L = grp_layout(KS);
    constexpr int NG = L.NG, MX = L.MHI, CW = 32 / NS;
    static_assert(NG <= 3, "the packed form serves KS <= 12");
    f32x2 y1[KS][1], e[NG][MX][1], A[NG][MX][1];
#pragma unroll
    for (int i = 0; i < KS; ++i) y1[i][0] = y[i];
    grp2_esp<KS, 0>(y1, e[0]);
    if constexpr (NG > 1) grp2_esp<KS, (NG > 1 ? 1 : 0)>(y1, e[NG > 1 ? 1 : 0]);
    if constexpr (NG > 2) grp2_esp<KS, (NG > 2 ? 2 : 0)>(y1, e[NG > 2 ? 2 : 0]);
#pragma unroll
    for (int gq = 0; gq < NG; ++gq)
#pragma unroll
        for (int j = 0; j < MX; ++j) A[gq][j][0] = 0ull;
    for (int p = 0; p < n_real; ++p, tab += ROWG) {                  // self-conjugate points
        float r[ROWG];
        load_row(tab, r);
        f32x2 q[NG], pre[NG];
#pragma unroll
        for (int gq = 0; gq < NG; ++gq) {
            const int Mg = grp_size(L, gq), co = gq < L.NHI ? 0 : ROWG_LO;
            f32x2 sacc = bcf(r[co]);
#pragma unroll
            for (int j = 0; j < MX; ++j)
                if (j < Mg) sacc = fma2(bcf(r[co + 2 * j + 2]), e[gq][j][0], sacc);
            q[gq] = sacc;
        }
        f32x2 run = q[0];
#pragma unroll
        for (int gq = 1; gq < NG; ++gq) { pre[gq] = run; run = mul2(run, q[gq]); }
        const f32x2 oth = shfl2(mask, run, CW);
        f32x2 suf = mul2(bcf(r[ROWG_W]), oth);
        fe = fma2(suf, run, fe);
        if (GRAD) {
#pragma unroll
            for (int gq = NG - 1; gq >= 0; --gq) {
                const int Mg = grp_size(L, gq), co = gq < L.NHI ? 0 : ROWG_LO;
                const f32x2 t = gq > 0 ? mul2(pre[gq], suf) : suf;
#pragma unroll
                for (int j = 0; j < MX; ++j)
                    if (j < Mg) A[gq][j][0] = fma2(bcf(r[co + 2 * j + 2]), t, A[gq][j][0]);
                if (gq > 0) suf = mul2(suf, q[gq]);
            }
        }
    }
    for (int p = 0; p < n_cplx; ++p, tab += ROWG) {                  // one of each conjugate pair
        float r[ROWG];
        load_row(tab, r);
        f32x2 qr[NG], qi[NG], nqi[NG], pr[NG], pi[NG];
#pragma unroll
        for (int gq = 0; gq < NG; ++gq) {
            const int Mg = grp_size(L, gq), co = gq < L.NHI ? 0 : ROWG_LO;
            f32x2 sr = bcf(r[co]), si = bcf(r[co + 1]);
#pragma unroll
            for (int j = 0; j < MX; ++j)
                if (j < Mg) { sr = fma2(bcf(r[co + 2 * j + 2]), e[gq][j][0], sr); si = fma2(bcf(r[co + 2 * j + 3]), e[gq][j][0], si); }
            qr[gq] = sr; qi[gq] = si; nqi[gq] = si ^ SGN2;
        }
        f32x2 rr = qr[0], ri = qi[0];
#pragma unroll
        for (int gq = 1; gq < NG; ++gq) {
            pr[gq] = rr; pi[gq] = ri;
            const f32x2 nr = fma2(rr, qr[gq], mul2(ri, nqi[gq]));     // Re: rr qr - ri qi
            const f32x2 ni = fma2(rr, qi[gq], mul2(ri, qr[gq]));      // Im: rr qi + ri qr
            rr = nr; ri = ni;
        }
        const f32x2 orr = shfl2(mask, rr, CW), oi = shfl2(mask, ri, CW);
        const float wr = r[ROWG_W], wi = r[ROWG_W + 1];
        f32x2 sr = fma2(bcf(wr), orr, mul2(bcf(-wi), oi)), si = fma2(bcf(wr), oi, mul2(bcf(wi), orr));   // suffix seeded with w x other
        fe = fma2(sr, rr, fe);
        fe = fma2(si ^ SGN2, ri, fe);                                 // Re(w other P_lane)
        if (GRAD) {
#pragma unroll
            for (int gq = NG - 1; gq >= 0; --gq) {
                const int Mg = grp_size(L, gq), co = gq < L.NHI ? 0 : ROWG_LO;
                f32x2 tr = sr, nti = si ^ SGN2;
                if (gq > 0) {
                    tr = fma2(pr[gq], sr, mul2(pi[gq], si ^ SGN2));   // Re: pr sr - pi si
                    nti = fma2(pr[gq], si, mul2(pi[gq], sr)) ^ SGN2;  // -Im
                }
#pragma unroll
                for (int j = 0; j < MX; ++j)
                    if (j < Mg) {
                        A[gq][j][0] = fma2(bcf(r[co + 2 * j + 2]), tr, A[gq][j][0]);
                        A[gq][j][0] = fma2(bcf(r[co + 2 * j + 3]), nti, A[gq][j][0]);     // Re(c_j T)
                    }
                if (gq > 0) {
                    const f32x2 nr = fma2(sr, qr[gq], mul2(si, nqi[gq]));
                    const f32x2 ni = fma2(sr, qi[gq], mul2(si, qr[gq]));
                    sr = nr; si = ni;
                }
            }
        }
    }
    if (GRAD) {
        f32x2 g1[KS][1];
#pragma unroll
        for (int i = 0; i < KS; ++i) g1[i][0] = 0ull;
        grp2_loo<KS, 0>(y1, A[0], g1);
        if constexpr (NG > 1) grp2_loo<KS, (NG > 1 ? 1 : 0)>(y1, A[NG > 1 ? 1 : 0], g1);
        if constexpr (NG > 2) grp2_loo<KS, (NG > 2 ? 2 : 0)>(y1, A[NG > 2 ? 2 : 0], g1);
#pragma unroll
        for (int i = 0; i < KS; ++i) g[i] = g1[i][0];
    }
}

template <int KS, int NS, bool GRAD>
__device__ __forceinline__ void run_item_split2(const EvalParams<float> &p, unsigned mask, const int32_t *__restrict__ s_lits,
                                                const float *__restrict__ s_tab, int n_real, int n_cplx, int nc, int wk,
                                                int h, int64_t b, f32x2 &fe, int k, float pad)
{
    const char *xb = reinterpret_cast<const char *>(p.x + b);
    char *gb = reinterpret_cast<char *>(p.G + (b - p.g_b0));
    const uint32_t x_ld = (uint32_t)(p.ldb * 4), g_ld = (uint32_t)(p.g_ld * 4);
    const int Wk = p.Wk;
    const bool miss = (KS - 1) * NS + h >= k;
    const f32x2 pad2 = pk(pad, pad);
    for (int c = wk; c < nc; c += Wk) {
        const int32_t *L = s_lits + c * k + h;
        int32_t lit[KS];
        f32x2 y[KS], g[KS];
#pragma unroll
        for (int i = 0; i < KS - 1; ++i) lit[i] = L[i * NS];
        lit[KS - 1] = miss ? LIT_NONE : L[(KS - 1) * NS];             // missing literal: constant, no gather, no RED
#pragma unroll
        for (int i = 0; i < KS; ++i) {
            f32x2 v[1] = {pad2};
            if (!(i == KS - 1 && (lit[i] & LIT_NONE)))
                PairIO<1>::load(xb + (uint64_t)(uint32_t)(lit[i] & LIT_VAR) * x_ld, v);
            const uint32_t m = (uint32_t)(lit[i] & LIT_NEG);
            y[i] = v[0] ^ (((f32x2)m << 32) | m);                     // y = s x (a missing slot: pad, its polarity bit is 0)
            g[i] = 0ull;
        }
        if (c + Wk < nc) {
            const int32_t *Ln = L + Wk * k;
#pragma unroll
            for (int i = 0; i < KS; ++i) {
                if (i == KS - 1 && miss) continue;
                const int32_t ln = Ln[i * NS];
                asm volatile("prefetch.global.L1 [%0];" ::"l"(xb + (uint64_t)(uint32_t)(ln & LIT_VAR) * x_ld));
            }
        }
        eval_points_grp2<KS, NS, GRAD>(mask, y, s_tab, n_real, n_cplx, fe, g);
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
__device__ __forceinline__ void item_body_split2(const EvalParams<float> &p, const int32_t *s_lits, const float *s_tab,
                                              float (*s_F)[64], int n_real, int n_cplx, int nc, int k, float pad)
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
        run_item_split2<KS, NS, GRAD>(p, mask, s_lits, s_tab, n_real, n_cplx, nc, wk, h, b, fe2, k, pad);
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
                                              T (*s_F)[32 * V], int n_real, int n_cplx, int nc, int k, T pad)
    {
        if (ks == KS) {
            if constexpr (V == 2) item_body_split2<KS, NS, GRAD>(p, s_lits, s_tab, s_F, n_real, n_cplx, nc, k, pad);
            else item_body_split<T, KS, NS, GRAD>(p, s_lits, s_tab, s_F, n_real, n_cplx, nc, k, pad);
        } else if (KS < KSHI)
            SwitchSplit<T, (KS < KSHI ? KS + 1 : KS), KSHI, NS, V, GRAD>::go(ks, p, s_lits, s_tab, s_F, n_real, n_cplx, nc, k, pad);
    }
};

// one launch for every length in [KLO, KHI]: the CTA's item picks the body compiled for ceil(k / NS) literals per lane.
// V = 1: scalar form; V = 2: packed form (fp32 only); both read the grouped staged table rowsg (ROWG scalars per point).
template <typename T, int KLO, int KHI, int NS, int V, bool GRAD, int THREADS, int MINB>
__global__ void __launch_bounds__(THREADS, MINB) k_eval_split(const EvalParams<T> p)
{
    __shared__ __align__(16) T s_tab[((KHI + 1) / 2 + 1) * ROWG];
    __shared__ int32_t s_lits[LIT_CHUNK];
    __shared__ T s_F[THREADS / 32][32 * V];
    const Item it = p.items[blockIdx.x];
    const SigDev sg = p.sigs[it.sig];
    const int nsc = (sg.n_real + sg.n_cplx) * ROWG;
    for (int i = threadIdx.x; i < nsc; i += blockDim.x) s_tab[i] = p.rowsg[(int64_t)sg.row2_off * ROWG + i];
    const int nl = (it.c_end - it.c_begin) * it.k;
    for (int i = threadIdx.x; i < nl; i += blockDim.x) s_lits[i] = __ldg(p.lits + it.lit_base + i);
    __syncthreads();
    SwitchSplit<T, (KLO + NS - 1) / NS, (KHI + NS - 1) / NS, NS, V, GRAD>::go((it.k + NS - 1) / NS, p, s_lits, s_tab, s_F, sg.n_real,
                                                                        sg.n_cplx, it.c_end - it.c_begin, it.k, (T)sg.pad);
}

#ifndef AFSAT_KS32_TU   // instantiated in afsat_ks32.cu
extern template __global__ void k_eval_split<float, AFSAT_L32_KMIN, AFSAT_MAX_LEN, AFSAT_L32_NS, 1, true, AFSAT_L32_THREADS, AFSAT_L32_MINB>(const EvalParams<float>);
extern template __global__ void k_eval_split<float, AFSAT_L32_KMIN, AFSAT_MAX_LEN, AFSAT_L32_NS, 1, false, AFSAT_L32_THREADS, AFSAT_L32_MINB>(const EvalParams<float>);
extern template __global__ void k_eval_split<double, AFSAT_L64_KMIN, AFSAT_MAX_LEN, 4, 1, true, AFSAT_L64_THREADS, 1>(const EvalParams<double>);
extern template __global__ void k_eval_split<double, AFSAT_L64_KMIN, AFSAT_MAX_LEN, 4, 1, false, AFSAT_L64_THREADS, 1>(const EvalParams<double>);
extern template __global__ void k_eval_split<double, AFSAT_A_KMAX + 1, AFSAT_B_KMAX, 2, 1, true, AFSAT_L64_THREADS, 1>(const EvalParams<double>);
extern template __global__ void k_eval_split<double, AFSAT_A_KMAX + 1, AFSAT_B_KMAX, 2, 1, false, AFSAT_L64_THREADS, 1>(const EvalParams<double>);
extern template __global__ void k_eval_split<float, AFSAT_A_KMAX + 1, AFSAT_B_KMAX, 2, 2, true, AFSAT_M32_THREADS, AFSAT_M32_MINB>(const EvalParams<float>);
extern template __global__ void k_eval_split<float, AFSAT_A_KMAX + 1, AFSAT_B_KMAX, 2, 2, false, AFSAT_M32_THREADS, AFSAT_M32_MINB>(const EvalParams<float>);
#endif

}  // namespace afsat
