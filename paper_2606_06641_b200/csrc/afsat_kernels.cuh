// afsat_kernels.cuh -- sm_100a device code of the AFSAT hot path.
//
// Mapping: LANE = V adjacent CANDIDATES.  X is variable-major [n][ldb], so
// the k literal gathers of a constraint are k coalesced, vectorised row segments per warp
// (LDG.64 for fp32, V = 2), the constraint's literal list / weight rows are warp-uniform (no
// divergence; they are staged once per work item in shared memory), and all prefix products live in
// registers.  A work item is a chunk of constraints of ONE signature (type, k, param); a CTA runs
// one item for Wc x (32 V) candidates, its Wk = warps/Wc warp groups interleaving the constraints.
//
// Per constraint and retained DFT point p the thread evaluates (afsat_host_tables)
//     f_i = a_p + b_p y_i,  P = prod_i f_i,  FE += Re(w_p P),
//     dFE/dy_i += Re( (w_p b_p) * prefix_{i-1} * suffix_{i+1} )        (leave-one-out, no division)
// and scatter-adds s_i dFE/dy_i into G[v_i][b..b+V) with one coalesced vector RED per literal.
//
// Sign rounding and the exact discrete count (a7, a8) never touch floating point beyond the one
// compare x < 0: k_update / k_pack_signs emit one bit per (variable, candidate) with a warp
// ballot, and k_check_bits counts true literals for 32 candidates at a time in bit-sliced integer
// arithmetic.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace afsat {

// packed literal: bits 0-29 variable, bit 31 negation (y = -x).  Fixed variables never reach a kernel: afsat_create
// substitutes them into the constraints.  LIT_NONE marks a literal slot a lane does not have
// (lane-split kernels, afsat_split.cuh).
constexpr int32_t LIT_NEG  = (int32_t)0x80000000u;
constexpr int32_t LIT_NONE = 0x40000000;
constexpr int32_t LIT_VAR  = 0x3FFFFFFF;

constexpr int LIT_CHUNK = 4096;       // packed literals staged in shared memory per work item
#define AFSAT_CTA_THREADS 256
constexpr int CTA_THREADS = AFSAT_CTA_THREADS;
constexpr int CTA_WARPS = CTA_THREADS / 32;
constexpr int MAX_ROWS = 33;          // retained DFT points per signature: H <= 64/2 + 1

struct SigDev {                 // 40 bytes, one per signature (type, k, param)
    int32_t row_off;            // first row in the weight table (8 scalars per row)
    int16_t n_real, n_cplx;     // real rows first, then complex rows
    uint64_t scan_lo, scan_hi;  // bit tau set: tau is in the SCANNED set of the discrete check
    int16_t scan_is_sat;        // 1: scanned set = satisfied counts; 0: = violated counts (smaller)
    int16_t chk_kind;           // k_check_bits: the predicate as a function of any / all / parity of the literals, or 0
    int32_t k;
    int32_t row2_off;           // first row of the STAGED table of the kernel that runs this length: rows2 (fp32, k <= 8,
                                // ROW2 scalars per row, pack_rows_f2) or rowsg (grouped lane-split kernels, pack_rows_grp)
    int8_t uv, n_unit, n_gen;   // rows2: unit variant, number of trivial-twiddle rows, number of generic complex rows
    int8_t pad;                 // rowsg: the literal value whose factor is exactly 1 (0 or 1)
    int32_t row2g_off, pad2;    // rows2g: first grouped generic row
};

struct Item {                   // one CTA-sized chunk of constraints of a single signature
    int32_t k, sig;
    int32_t c_begin, c_end;     // constraint range in bucket order
    int64_t lit_base;           // offset of c_begin's first packed literal
    int32_t pad0, pad1;
};

template <typename T>
struct EvalParams {
    const T *x;                 // [n][ldb]
    T *G;                       // gradient accumulator (RED; zero on entry) or null
    int64_t g_ld;               // leading dimension of G (ldb, or the tile width of the scratch)
    int64_t g_b0;               // G column of candidate b is (b - g_b0)
    T *Fpart;                   // [n_frows][ldb] per-(item, warp group) partial objective or null
    const int32_t *lits;        // packed literals, bucket order
    const SigDev *sigs;
    const T *rows;              // weight table
    const float *rows2;         // staged table of the packed fp32 kernel (fp32 contexts), else null
    const float *rows2g;        // packed fp32 kernel: the generic complex rows staged for literal groups (ROW2G scalars per row)
    const T *rowsg;             // staged table of the grouped lane-split kernels (afsat_split.cuh), ROWG scalars per row
    const Item *items;          // items of this launch
    int32_t frow_base;          // row of Fpart for (items[0], group 0)
    int32_t B;
    int64_t ldb;
    int64_t b_begin, b_end;     // candidate tile of this launch (b_end <= ldb)
    int32_t Wc, Wk;             // warps of a CTA: Wc candidate sub-tiles x Wk constraint groups
    int32_t cs;                 // k_eval_f2m: a warp's lanes take cs (1, 2 or 4) constraints at once, 32 / cs lanes each
    const uint8_t *skip;        // [ldb] or null: candidates with skip[b] != 0 are not evaluated (line search)
};

// lane-level test of the skip mask for the V candidates b .. b+V-1 of a lane (all must be skipped)
template <typename T>
__device__ __forceinline__ bool lane_skipped(const EvalParams<T> &p, int64_t b, int V)
{
    if (!p.skip) return false;
    bool all = true;
    for (int v = 0; v < V; ++v) all = all && (b + v >= p.ldb || p.skip[b + v] != 0);
    return all;
}

template <typename T> __device__ __forceinline__ T fma_(T a, T b, T c);
template <> __device__ __forceinline__ float fma_<float>(float a, float b, float c) { return fmaf(a, b, c); }
template <> __device__ __forceinline__ double fma_<double>(double a, double b, double c) { return fma(a, b, c); }

// ---- vector gather / vector RED ------------------------------------------------------------------
// scalar RED as inline PTX: atomicAdd on a pointer the compiler cannot prove global compiles to ATOM plus a
// shared-window test with a CAS fallback
__device__ __forceinline__ void red_add(float *p, float v) { asm volatile("red.global.add.f32 [%0], %1;" ::"l"(p), "f"(v) : "memory"); }
__device__ __forceinline__ void red_add(double *p, double v) { asm volatile("red.global.add.f64 [%0], %1;" ::"l"(p), "d"(v) : "memory"); }
template <typename T, int V> struct VecIO;
template <> struct VecIO<float, 1> {
    static __device__ __forceinline__ void load(const float *p, float (&v)[1]) { v[0] = __ldg(p); }
    static __device__ __forceinline__ void red(float *p, const float (&v)[1]) { red_add(p, v[0]); }
};
template <> struct VecIO<float, 2> {
    static __device__ __forceinline__ void load(const float *p, float (&v)[2])
    {
        const float2 t = __ldg(reinterpret_cast<const float2 *>(p));
        v[0] = t.x; v[1] = t.y;
    }
    static __device__ __forceinline__ void red(float *p, const float (&v)[2])
    {
        asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" ::"l"(p), "f"(v[0]), "f"(v[1]) : "memory");
    }
};
template <> struct VecIO<float, 4> {
    static __device__ __forceinline__ void load(const float *p, float (&v)[4])
    {
        const float4 t = __ldg(reinterpret_cast<const float4 *>(p));
        v[0] = t.x; v[1] = t.y; v[2] = t.z; v[3] = t.w;
    }
    static __device__ __forceinline__ void red(float *p, const float (&v)[4])
    {
        asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(v[0]), "f"(v[1]), "f"(v[2]), "f"(v[3])
                     : "memory");
    }
};
template <> struct VecIO<double, 1> {
    static __device__ __forceinline__ void load(const double *p, double (&v)[1]) { v[0] = __ldg(p); }
    static __device__ __forceinline__ void red(double *p, const double (&v)[1]) { red_add(p, v[0]); }
};
template <> struct VecIO<double, 2> {
    static __device__ __forceinline__ void load(const double *p, double (&v)[2])
    {
        const double2 t = __ldg(reinterpret_cast<const double2 *>(p));
        v[0] = t.x; v[1] = t.y;
    }
    static __device__ __forceinline__ void red(double *p, const double (&v)[2])
    {
        red_add(p, v[0]); red_add(p + 1, v[1]);
    }
};

// ---- a2-a4 for one constraint of compile-time length K and V candidates, all in registers --------
// tab: the signature's rows in shared memory, 8 scalars per row {Re a, Im a, Re b, Im b, Re w, Im w,
// Re(w b), Im(w b)}, real rows first.
template <typename T, int K, int V, bool GRAD>
__device__ __forceinline__ void eval_points_reg(const T (&y)[K][V], const T *__restrict__ tab, int n_real,
                                                int n_cplx, T (&fe)[V], T (&g)[K][V])
{
    const T *r = tab;
    for (int p = 0; p < n_real; ++p, r += 8) {                       // self-conjugate points
        const T a = r[0], b = r[2], w = r[4], wb = r[6];
#pragma unroll
        for (int v = 0; v < V; ++v) {
            T pre[K], f[K];
#pragma unroll
            for (int i = 0; i < K; ++i) f[i] = fma_(b, y[i][v], a);
            T run = f[0];
#pragma unroll
            for (int i = 1; i < K; ++i) { pre[i] = run; run *= f[i]; }
            fe[v] = fma_(w, run, fe[v]);
            if (GRAD) {
                T suf = wb;
#pragma unroll
                for (int i = K - 1; i >= 1; --i) { g[i][v] = fma_(pre[i], suf, g[i][v]); suf *= f[i]; }
                g[0][v] += suf;                                       // prefix_0 = 1
            }
        }
    }
    for (int p = 0; p < n_cplx; ++p, r += 8) {                       // one of each conjugate pair
        const T ar = r[0], ai = r[1], br = r[2], bi = r[3], wr = r[4], wi = r[5], wbr = r[6], wbi = r[7];
#pragma unroll
        for (int v = 0; v < V; ++v) {
            T pr[K], pi[K], fr[K], fi[K];
#pragma unroll
            for (int i = 0; i < K; ++i) { fr[i] = fma_(br, y[i][v], ar); fi[i] = fma_(bi, y[i][v], ai); }
            T rr = fr[0], ri = fi[0];
#pragma unroll
            for (int i = 1; i < K; ++i) {
                pr[i] = rr; pi[i] = ri;
                const T nr = fma_(rr, fr[i], -(ri * fi[i]));
                const T ni = fma_(rr, fi[i], ri * fr[i]);
                rr = nr; ri = ni;
            }
            fe[v] = fma_(wr, rr, fe[v]);
            fe[v] = fma_(-wi, ri, fe[v]);
            if (GRAD) {
                T sr = wbr, si = wbi;                                 // suffix seeded with w b
#pragma unroll
                for (int i = K - 1; i >= 1; --i) {
                    g[i][v] = fma_(pr[i], sr, g[i][v]);
                    g[i][v] = fma_(-pi[i], si, g[i][v]);
                    const T nr = fma_(sr, fr[i], -(si * fi[i]));
                    const T ni = fma_(sr, fi[i], si * fr[i]);
                    sr = nr; si = ni;
                }
                g[0][v] += sr;                                        // prefix_0 = 1
            }
        }
    }
}

// ---- packed fp32 pairs (sm_100a FFMA2): one instruction evaluates BOTH candidates of a lane ---------
// fma.rn.f32x2 issues at half the rate of FFMA but does two FMAs, so the FP32 pipe stays the bound
// while the issue slots freed carry the integer / load-store overhead (measured: DESIGN.md "FFMA2").
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk(float lo, float hi)
{
    f32x2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r;
}
__device__ __forceinline__ void upk(f32x2 v, float &lo, float &hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c)
{
    f32x2 d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b)
{
    f32x2 d; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d;
}
// pair (c, c) from entry j of a packed table, read as ONE scalar so that the compiler can use the
// broadcast operand form
__device__ __forceinline__ f32x2 bc(const f32x2 *tab, int j)
{
    const float c = reinterpret_cast<const float *>(tab)[2 * j];
    return pk(c, c);
}
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b)
{
    f32x2 d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d;
}

// Rows of the packed table in shared memory: 12 pairs (c, c) per DFT point.
//   real point:    {a, b, w, wb, -, -, -, -, -, -, -, -}
//   complex point: {ar, ai, -ai, br, bi, -bi, wr, -wi, Re(wb), -Im(wb), -, -}
// FFMA2 has no negated operands, so the negated imaginary parts are tabulated and the backward
// walk carries the suffix as (Re s, -Im s).
constexpr int ROW2 = 12;
#define AFSAT_PACK_MAX_ROWS 40              // >= MAX_ROWS + the zero-weight unit rows a table may get


// HOST: the staged table of one signature for the packed kernel, from its fp32 rows {Re a, Im a, Re b, Im b,
// Re w, Im w, Re(wb), Im(wb)} (real rows first).  Standard tables (a = 1/2 exactly in every row): the
// trivial twiddles first, at fixed positions -- [w = 1 (absent: uv = 2)] [w = -1 iff k odd] [w = i iff k = 3] -- a missing
// one (its weight was exactly zero) staged with weight 0, the halvings folded into their weights (2^-k, 2^-(k-1): exact
// rescales); then the complex rows, which run the literal groups.  (k = 7 has the points i and the eighth roots, which
// rounds 1 and 2 walked on their own, two adds and two FMAs per multiplication: with the weight folded into the
// coefficients and the contraction read off the accumulators the grouped rows are the cheaper form for them too, cfg1
// 1.79 -> 1.68 ms per step with the objective.)  Other tables: rows as they are, uv = 0.
// The generic complex rows are ALSO staged for literal groups (grp_rows_f2; outg gets ROW2G scalars per generic row, rd are
// the same rows in double): c_j = a^(M-j) b^j for the two group sizes, and w c_j (as Re, -Im) beside them; for the standard
// tables un-halved (a = 1, b = w^l, the 2^-k folded into the weight: exact rescales).
// Returns the number of staged rows; out gets ROW2 scalars per row.
constexpr int ROW2G_G1_H = 10, ROW2G_D0_H = 20, ROW2G_D1_H = 30, ROW2G_H = 40;    // = ROW2G_G1, ROW2G_D0, ROW2G_D1, ROW2G below
inline int pack_rows_f2(const float *r0, const double *rd, int n_real, int n_cplx, int k, float *out, float *outg, int *uv_out,
                        int *n_unit_out, int *n_gen_out)
{
    const int nr = n_real + n_cplx;
    int src[AFSAT_PACK_MAX_ROWS], n = 0, uv = 0, n_unit = n_real, n_gen = n_cplx;
    bool std_tab = true;
    for (int q = 0; q < nr; ++q) std_tab = std_tab && r0[8 * q] == 0.5f && r0[8 * q + 1] == 0.f;
    if (std_tab) {
        int iP = -1, iM = -1, iI = -1;
        for (int q = 0; q < nr; ++q) {
            const float br = r0[8 * q + 2], bi = r0[8 * q + 3];
            if (q < n_real) { if (br == 0.5f) iP = q; else if (br == -0.5f) iM = q; }
            else if (k == 3 && br == 0.f && bi == 0.5f) iI = q;
        }
        uv = iP >= 0 ? 1 : 2;
        if (iP >= 0) src[n++] = iP;
        if (k & 1) src[n++] = iM;
        if (k == 3) src[n++] = iI;
        n_unit = n;
        for (int q = n_real; q < nr; ++q) if (q != iI) src[n++] = q;
        n_gen = n - n_unit;
    } else {
        for (int q = 0; q < nr; ++q) src[n++] = q;
    }
    float sc_w = 1.f;
    for (int i = 0; i < k; ++i) sc_w *= 0.5f;                                   // 2^-k
    const float sc_wb = 2.0f * sc_w;                                            // 2^-(k-1)
    for (int q = 0; q < n; ++q) {
        float *o = out + (size_t)q * ROW2;
        for (int j = 0; j < ROW2; ++j) o[j] = 0.f;
        if (src[q] < 0) continue;
        const float *r = r0 + 8 * src[q];
        const bool unit = uv != 0 && q < n_unit;
        const float fw = unit ? sc_w : 1.f, fwb = unit ? sc_wb : 1.f;
        if (src[q] < n_real) { o[0] = r[0]; o[1] = r[2]; o[2] = r[4] * fw; o[3] = r[6] * fwb; }   // a, b, w, wb
        else {
            o[0] = r[0]; o[1] = r[1]; o[2] = -r[1]; o[3] = r[2]; o[4] = r[3]; o[5] = -r[3];
            o[6] = r[4] * fw; o[7] = -r[5] * fw; o[8] = r[6] * fwb; o[9] = -r[7] * fwb;
        }
    }
    {
        const int M[2] = {(k + 1) / 2, k / 2}, off[2] = {0, ROW2G_G1_H}, offd[2] = {ROW2G_D0_H, ROW2G_D1_H};
        double scw = 1.0;
        if (std_tab) for (int i = 0; i < k; ++i) scw *= 0.5;
        const double sc = std_tab ? 2.0 : 1.0;
        for (int q = n_unit; q < n; ++q) {
            float *o = outg + (size_t)(q - n_unit) * ROW2G_H;
            for (int j = 0; j < ROW2G_H; ++j) o[j] = 0.f;
            const double *r = rd + 8 * src[q];
            const double ar = sc * r[0], ai = sc * r[1], br = sc * r[2], bi = sc * r[3];
            for (int gq = 0; gq < 2; ++gq)
                for (int j = 0; j <= M[gq]; ++j) {
                    double cr = 1.0, ci = 0.0;
                    for (int t = 0; t < M[gq]; ++t) {
                        const double fr = t < j ? br : ar, fi = t < j ? bi : ai;
                        const double nr2 = cr * fr - ci * fi, ni2 = cr * fi + ci * fr;
                        cr = nr2; ci = ni2;
                    }
                    o[off[gq] + 2 * j] = (float)cr; o[off[gq] + 2 * j + 1] = (float)ci;
                    // the same coefficient times the point's weight, as (Re, -Im): sum_j (w c_j) e_j = w x (the group's factor)
                    const double wr = r[4] * scw, wi = r[5] * scw;
                    o[offd[gq] + 2 * j] = (float)(wr * cr - wi * ci); o[offd[gq] + 2 * j + 1] = (float)-(wr * ci + wi * cr);
                }
        }
    }
    *uv_out = uv; *n_unit_out = n_unit; *n_gen_out = n_gen;
    return n;
}

constexpr f32x2 NEGP = 0x8000000080000000ull;

// ---- trivial twiddles (standard tables only: a = 1/2 exactly) ---------------------------------------
// With the halving folded into the weights (w 2^-k, w b 2^-(k-1): exact power-of-two rescales done when
// the row is staged) a factor is 1 + (b/a) y, and for the DFT points w^l in {1, -1, i} -- l = 0, N/2, N/4,
// the twiddles every FFT treats as free -- the product needs no multiplication by a coefficient:
//   real:  P <- P + P y'                      (y' = y or -y)                1 FFMA2 per literal
//   w = i: P <- (Re P - y Im P) + i (Im P + y Re P)                         2 FFMA2 per literal

// The unit rows of a signature are walked TOGETHER (HP: w = 1, HM: w = -1, HI: w = i): each is a serial
// chain of dependent FFMA2s, so interleaving them is what keeps the FMA pipe fed at 4 warps per scheduler.
template <int K, int NP, bool HP, bool HM, bool HI, int GRAD>
__device__ __forceinline__ void unit_rows_f2(const f32x2 (&y)[K][NP], const f32x2 *__restrict__ rP, const f32x2 *__restrict__ rM,
                                             const f32x2 *__restrict__ rI, f32x2 (&fe)[NP], f32x2 (&g)[K][NP])
{
    const f32x2 one2 = pk(1.0f, 1.0f);
    f32x2 ny[K][NP], preP[HP ? K : 1][NP], preM[HM ? K : 1][NP], pr[HI ? K : 1][NP], pi[HI ? K : 1][NP];
    f32x2 runP[NP], runM[NP], rr[NP], ri[NP];
#pragma unroll
    for (int i = 0; i < K; ++i)
#pragma unroll
        for (int q = 0; q < NP; ++q) ny[i][q] = y[i][q] ^ NEGP;
#pragma unroll
    for (int q = 0; q < NP; ++q) {
        if (HP) runP[q] = add2(y[0][q], one2);                                       // 1 + y_0
        if (HM) runM[q] = add2(ny[0][q], one2);                                      // 1 - y_0
        if (HI) { rr[q] = one2; ri[q] = y[0][q]; }                                   // 1 + i y_0
    }
#pragma unroll
    for (int i = 1; i < K; ++i)
#pragma unroll
        for (int q = 0; q < NP; ++q) {
            if (HP) { preP[i][q] = runP[q]; runP[q] = fma2(runP[q], y[i][q], runP[q]); }
            if (HM) { preM[i][q] = runM[q]; runM[q] = fma2(runM[q], ny[i][q], runM[q]); }
            if (HI) {
                pr[i][q] = rr[q]; pi[i][q] = ri[q];
                const f32x2 nr = fma2(ny[i][q], ri[q], rr[q]);                       // Re: rr - y ri
                const f32x2 ni = fma2(y[i][q], rr[q], ri[q]);                        // Im: ri + y rr
                rr[q] = nr; ri[q] = ni;
            }
        }
#pragma unroll
    for (int q = 0; q < NP; ++q) {
        if (GRAD == 2) break;                                                        // gradient only
        if (HP) fe[q] = fma2(bc(rP, 2), runP[q], fe[q]);
        if (HM) fe[q] = fma2(bc(rM, 2), runM[q], fe[q]);
        if (HI) { fe[q] = fma2(bc(rI, 6), rr[q], fe[q]); fe[q] = fma2(bc(rI, 7), ri[q], fe[q]); }   // + wr Re P - wi Im P
    }
    if (GRAD) {
        f32x2 sufP[NP], sufM[NP], sr[NP], nsi[NP];                                   // suffixes seeded with w b; (Re s, -Im s)
#pragma unroll
        for (int q = 0; q < NP; ++q) {
            if (HP) sufP[q] = bc(rP, 3);
            if (HM) sufM[q] = bc(rM, 3);
            if (HI) { sr[q] = rI[8]; nsi[q] = rI[9]; }
        }
#pragma unroll
        for (int i = K - 1; i >= 1; --i)
#pragma unroll
            for (int q = 0; q < NP; ++q) {
                if (HP) { g[i][q] = fma2(preP[i][q], sufP[q], g[i][q]); sufP[q] = fma2(sufP[q], y[i][q], sufP[q]); }
                if (HM) { g[i][q] = fma2(preM[i][q], sufM[q], g[i][q]); sufM[q] = fma2(sufM[q], ny[i][q], sufM[q]); }
                if (HI) {
                    g[i][q] = fma2(pr[i][q], sr[q], g[i][q]);                        // Re(pre suf) = pr sr - pi si
                    g[i][q] = fma2(pi[i][q], nsi[q], g[i][q]);
                    const f32x2 t_r = fma2(y[i][q], nsi[q], sr[q]);                  // Re: sr - y si
                    const f32x2 t_n = fma2(ny[i][q], sr[q], nsi[q]);                 // -Im: -(si + y sr)
                    sr[q] = t_r; nsi[q] = t_n;
                }
            }
#pragma unroll
        for (int q = 0; q < NP; ++q) {                                               // prefix_0 = 1
            if (HP) g[0][q] = add2(g[0][q], sufP[q]);
            if (HM) g[0][q] = add2(g[0][q], sufM[q]);
            if (HI) g[0][q] = add2(g[0][q], sr[q]);
        }
    }
}

// ---- literal GROUPS at the generic complex DFT points (packed form) ---------------------------------------------------
// The product of M factors is the polynomial  prod_{u<M} (a + b y_u) = sum_{j<=M} a^(M-j) b^j e_j(y_group)  in the group's
// elementary symmetric polynomials, which do not depend on the DFT point: they are formed once per constraint, and at
// every point a group costs 2 M FFMA2 for its complex factor (coefficients through the broadcast operand) instead of M
// factors and M - 1 complex multiplies.  The partial gradients come out of M accumulators per group,
//     A_j += Re( w a^(M-j) b^j x (product of the OTHER groups' factors) ),   dFE/dy_u = sum_j A_j e_{j-1}(group without y_u),
// expanded once per constraint.  The generating polynomial is still evaluated at every DFT point and contracted with the
// same weights; the groups only change the order in which its factors are multiplied.
__device__ __forceinline__ f32x2 bcf(float c) { return pk(c, c); }

// e[j-1] = e_j(y[0..M)), M <= 4
template <int M, int NP>
__device__ __forceinline__ void esp_f2(const f32x2 (*y)[NP], f32x2 (&e)[M][NP])
{
    static_assert(M >= 1 && M <= 4, "group size");
#pragma unroll
    for (int q = 0; q < NP; ++q) {
        if (M == 1) { e[0][q] = y[0][q]; }
        else if (M == 2) { e[0][q] = add2(y[0][q], y[1][q]); e[M > 1 ? 1 : 0][q] = mul2(y[0][q], y[M > 1 ? 1 : 0][q]); }
        else if (M == 3) {
            const f32x2 s01 = add2(y[0][q], y[1][q]), p01 = mul2(y[0][q], y[1][q]), y2 = y[M > 2 ? 2 : 0][q];
            e[0][q] = add2(s01, y2); e[M > 1 ? 1 : 0][q] = fma2(s01, y2, p01); e[M > 2 ? 2 : 0][q] = mul2(p01, y2);
        } else {
            const f32x2 s01 = add2(y[0][q], y[1][q]), p01 = mul2(y[0][q], y[1][q]);
            const f32x2 s23 = add2(y[M > 2 ? 2 : 0][q], y[M > 3 ? 3 : 0][q]), p23 = mul2(y[M > 2 ? 2 : 0][q], y[M > 3 ? 3 : 0][q]);
            e[0][q] = add2(s01, s23);
            e[M > 1 ? 1 : 0][q] = fma2(s01, s23, add2(p01, p23));
            e[M > 2 ? 2 : 0][q] = fma2(p01, s23, mul2(p23, s01));
            e[M > 3 ? 3 : 0][q] = mul2(p01, p23);
        }
    }
}

// g[u] += sum_j A[j] e_j(y without y_u), j = 0 .. M-1
template <int M, int NP>
__device__ __forceinline__ void loo_f2(const f32x2 (*y)[NP], const f32x2 (&A)[M][NP], f32x2 (*g)[NP])
{
#pragma unroll
    for (int q = 0; q < NP; ++q) {
        if (M == 1) { g[0][q] = add2(g[0][q], A[0][q]); }
        else if (M == 2) {
            g[0][q] = add2(g[0][q], fma2(A[M > 1 ? 1 : 0][q], y[M > 1 ? 1 : 0][q], A[0][q]));
            g[M > 1 ? 1 : 0][q] = add2(g[M > 1 ? 1 : 0][q], fma2(A[M > 1 ? 1 : 0][q], y[0][q], A[0][q]));
        } else if (M == 3) {
            const f32x2 y0 = y[0][q], y1 = y[M > 1 ? 1 : 0][q], y2 = y[M > 2 ? 2 : 0][q];
            const f32x2 a0 = A[0][q], a1 = A[M > 1 ? 1 : 0][q], a2 = A[M > 2 ? 2 : 0][q];
            g[0][q] = add2(g[0][q], fma2(a2, mul2(y1, y2), fma2(a1, add2(y1, y2), a0)));
            g[M > 1 ? 1 : 0][q] = add2(g[M > 1 ? 1 : 0][q], fma2(a2, mul2(y0, y2), fma2(a1, add2(y0, y2), a0)));
            g[M > 2 ? 2 : 0][q] = add2(g[M > 2 ? 2 : 0][q], fma2(a2, mul2(y0, y1), fma2(a1, add2(y0, y1), a0)));
        } else {
            const f32x2 y0 = y[0][q], y1 = y[M > 1 ? 1 : 0][q], y2 = y[M > 2 ? 2 : 0][q], y3 = y[M > 3 ? 3 : 0][q];
            const f32x2 a0 = A[0][q], a1 = A[M > 1 ? 1 : 0][q], a2 = A[M > 2 ? 2 : 0][q], a3 = A[M > 3 ? 3 : 0][q];
            const f32x2 s01 = add2(y0, y1), p01 = mul2(y0, y1), s23 = add2(y2, y3), p23 = mul2(y2, y3);
            // others of y0: {y1, y2, y3}: e1 = y1 + s23, e2 = y1 s23 + p23, e3 = y1 p23; and so on
            g[0][q] = add2(g[0][q], fma2(a3, mul2(y1, p23), fma2(a2, fma2(y1, s23, p23), fma2(a1, add2(y1, s23), a0))));
            g[M > 1 ? 1 : 0][q] = add2(g[M > 1 ? 1 : 0][q], fma2(a3, mul2(y0, p23), fma2(a2, fma2(y0, s23, p23), fma2(a1, add2(y0, s23), a0))));
            g[M > 2 ? 2 : 0][q] = add2(g[M > 2 ? 2 : 0][q], fma2(a3, mul2(y3, p01), fma2(a2, fma2(y3, s01, p01), fma2(a1, add2(y3, s01), a0))));
            g[M > 3 ? 3 : 0][q] = add2(g[M > 3 ? 3 : 0][q], fma2(a3, mul2(y2, p01), fma2(a2, fma2(y2, s01, p01), fma2(a1, add2(y2, s01), a0))));
        }
    }
}

// Staged row of a generic complex point for TWO groups (sizes M0 = ceil(K/2), M1 = floor(K/2) <= 4): {Re, Im of c0_0 ..
// c0_M0 | Re, Im of c1_0 .. c1_M1 (from scalar ROW2G_G1) | Re, -Im of w c0_j (ROW2G_D0) | Re, -Im of w c1_j (ROW2G_D1)},
// c_j = a^(M-j) b^j of the group, w the point's contracted weight.
constexpr int ROW2G_G1 = ROW2G_G1_H, ROW2G_D0 = ROW2G_D0_H, ROW2G_D1 = ROW2G_D1_H, ROW2G = ROW2G_H;

// all generic complex rows of a signature for the K literals of a lane (K >= 2), two groups
// ROLLED: the loop over the DFT points is kept as it is written (the compiler's two-fold unrolling pays for itself with a
// dozen register-renaming moves per constraint: with four candidates per lane cfg4 17.38 -> 17.2 ms per step; with two
// candidates per lane the unrolled form is the faster one, cfg1)
template <int K, int NP, int GRAD, bool ROLLED>
__device__ __forceinline__ void grp_rows_f2_joint(const f32x2 (&y)[K][NP], const float *__restrict__ rg, int n_rows, f32x2 (&fe)[NP],
                                            f32x2 (&g)[K][NP])
{
    constexpr int M0 = (K + 1) / 2, M1 = K / 2;
    f32x2 e0[M0][NP], e1[M1][NP], A0[M0][NP], A1[M1][NP], A00[NP];
    esp_f2<M0, NP>(&y[0], e0);
    esp_f2<M1, NP>(&y[M0], e1);
#pragma unroll
    for (int q = 0; q < NP; ++q) {
#pragma unroll
        for (int j = 0; j < M0; ++j) A0[j][q] = 0ull;
#pragma unroll
        for (int j = 0; j < M1; ++j) A1[j][q] = 0ull;
        A00[q] = 0ull;
    }
    // Per point, with the weight folded into a second set of coefficients on the host: T0 = w q1 = sum_j (w c1_j) e1_j is
    // everything but group 0, T1 = w q0 everything but group 1 -- each costs what the bare factor costs, and the four
    // packed multiplications by w of the earlier form are gone.  A_j += Re(c_j T) = Re c_j Re T - Im c_j Im T;
    // the contraction a3 is Re(w P) = Re(T0 q0) and needs the bare q0 (GRAD != 2 only).
    auto row = [&](const float *__restrict__ rg) {
#pragma unroll
        for (int q = 0; q < NP; ++q) {
            f32x2 t0r = bcf(rg[ROW2G_D1]), nt0i = bcf(rg[ROW2G_D1 + 1]);
#pragma unroll
            for (int j = 0; j < M1; ++j) {
                t0r = fma2(bcf(rg[ROW2G_D1 + 2 + 2 * j]), e1[j][q], t0r); nt0i = fma2(bcf(rg[ROW2G_D1 + 3 + 2 * j]), e1[j][q], nt0i);
            }
            if (GRAD == 0) {
                f32x2 q0r = bcf(rg[0]), q0i = bcf(rg[1]);
#pragma unroll
                for (int j = 0; j < M0; ++j) { q0r = fma2(bcf(rg[2 + 2 * j]), e0[j][q], q0r); q0i = fma2(bcf(rg[3 + 2 * j]), e0[j][q], q0i); }
                fe[q] = fma2(t0r, q0r, fe[q]);
                fe[q] = fma2(nt0i, q0i, fe[q]);                       // Re(T0 q0)
            }
            if (GRAD == 1) {                                          // the constant term of group 0: see below
                A00[q] = fma2(bcf(rg[0]), t0r, A00[q]); A00[q] = fma2(bcf(rg[1]), nt0i, A00[q]);
            }
            if (GRAD) {
                f32x2 t1r = bcf(rg[ROW2G_D0]), nt1i = bcf(rg[ROW2G_D0 + 1]);
#pragma unroll
                for (int j = 0; j < M0; ++j) {
                    t1r = fma2(bcf(rg[ROW2G_D0 + 2 + 2 * j]), e0[j][q], t1r); nt1i = fma2(bcf(rg[ROW2G_D0 + 3 + 2 * j]), e0[j][q], nt1i);
                }
#pragma unroll
                for (int j = 0; j < M0; ++j) {
                    A0[j][q] = fma2(bcf(rg[2 + 2 * j]), t0r, A0[j][q]); A0[j][q] = fma2(bcf(rg[3 + 2 * j]), nt0i, A0[j][q]);
                }
#pragma unroll
                for (int j = 0; j < M1; ++j) {
                    A1[j][q] = fma2(bcf(rg[ROW2G_G1 + 2 + 2 * j]), t1r, A1[j][q]);
                    A1[j][q] = fma2(bcf(rg[ROW2G_G1 + 3 + 2 * j]), nt1i, A1[j][q]);
                }
            }
        }
    };
    if constexpr (ROLLED) {
#pragma unroll 1
        for (int p = 0; p < n_rows; ++p, rg += ROW2G) row(rg);
    } else {
        for (int p = 0; p < n_rows; ++p, rg += ROW2G) row(rg);
    }
    if (GRAD == 1) {
        // The contraction a3 out of the gradient's accumulators: at every point Re(w P) = Re(T0 q0) is LINEAR in group 0's
        // symmetric polynomials, q0 = c0_0 + sum_j c0_j e_j, so summed over the points FE = A0_0 + sum_j A0_j e_j with
        // A0_j = sum_points Re(c0_j T0) -- the accumulators of the gradient plus one for the constant term.
#pragma unroll
        for (int q = 0; q < NP; ++q) {
            f32x2 f = A00[q];
#pragma unroll
            for (int j = 0; j < M0; ++j) f = fma2(A0[j][q], e0[j][q], f);
            fe[q] = add2(fe[q], f);
        }
    }
    if (GRAD) {
        loo_f2<M0, NP>(&y[0], A0, &g[0]);
        loo_f2<M1, NP>(&y[M0], A1, &g[M0]);
    }
}

// With two pairs per lane and K >= AFSAT_F2_SEQ_MINK the pairs are walked one after the other (each keeps ~4 K register
// pairs of symmetric polynomials, accumulators and literal values alive).
#define AFSAT_F2_SEQ_MINK 5
template <int K, int NP, int GRAD>
__device__ __forceinline__ void grp_rows_f2(const f32x2 (&y)[K][NP], const float *__restrict__ rg, int n_rows, f32x2 (&fe)[NP],
                                            f32x2 (&g)[K][NP])
{
    if constexpr (NP == 1 || K < AFSAT_F2_SEQ_MINK) {
        grp_rows_f2_joint<K, NP, GRAD, NP == 2>(y, rg, n_rows, fe, g);
    } else {
#pragma unroll
        for (int q = 0; q < NP; ++q) {
            f32x2 y1[K][1], g1[K][1], fe1[1];
#pragma unroll
            for (int i = 0; i < K; ++i) { y1[i][0] = y[i][q]; g1[i][0] = g[i][q]; }
            fe1[0] = fe[q];
            grp_rows_f2_joint<K, 1, GRAD, true>(y1, rg, n_rows, fe1, g1);
#pragma unroll
            for (int i = 0; i < K; ++i) g[i][q] = g1[i][0];
            fe[q] = fe1[0];
        }
    }
}

// UV (unit variant, chosen once per work item when its table is staged): 0 = generic coefficients in
// every row; 1 / 2 = standard table whose first rows are the trivial twiddles [w = 1 (UV 1 only)]
// [w = -1 iff K odd] [w = i iff K = 3] (n_real = their number), followed by n_cplx complex rows for the literal groups.
template <int K, int NP, int GRAD, int UV>
__device__ __forceinline__ void eval_points_f2(const f32x2 (&y)[K][NP], const f32x2 *__restrict__ tab, const float *__restrict__ tabg,
                                               int n_real, int n_cplx, f32x2 (&fe)[NP], f32x2 (&g)[K][NP])
{
    if (UV != 0) {
        constexpr bool HP = UV == 1, HM = (K & 1) != 0, HI = K == 3;
        const f32x2 *rP = tab, *rM = tab + (HP ? ROW2 : 0), *rI = rM + (HM ? ROW2 : 0);
        if (HP || HM || HI) unit_rows_f2<K, NP, HP, HM, HI, GRAD>(y, rP, rM, rI, fe, g);
        // the other complex points, grouped (K = 3 has none: its one complex point is w = i)
        if constexpr (K >= 2 && K != 3) { if (n_cplx > 0) grp_rows_f2<K, NP, GRAD>(y, tabg, n_cplx, fe, g); }
        return;
    }
    const f32x2 *r = tab;
    for (int p = 0; p < n_real; ++p, r += ROW2) {                    // self-conjugate points, generic coefficients
        const f32x2 a = bc(r, 0), b = bc(r, 1), w = bc(r, 2), wb = bc(r, 3);
        f32x2 pre[K][NP], f[K][NP], run[NP], suf[NP];
#pragma unroll
        for (int i = 0; i < K; ++i)
#pragma unroll
            for (int q = 0; q < NP; ++q) f[i][q] = fma2(b, y[i][q], a);
#pragma unroll
        for (int q = 0; q < NP; ++q) run[q] = f[0][q];
#pragma unroll
        for (int i = 1; i < K; ++i)
#pragma unroll
            for (int q = 0; q < NP; ++q) { pre[i][q] = run[q]; run[q] = mul2(run[q], f[i][q]); }
#pragma unroll
        for (int q = 0; q < NP; ++q) if (GRAD != 2) fe[q] = fma2(w, run[q], fe[q]);
        if (GRAD) {
#pragma unroll
            for (int q = 0; q < NP; ++q) suf[q] = wb;
#pragma unroll
            for (int i = K - 1; i >= 1; --i)
#pragma unroll
                for (int q = 0; q < NP; ++q) { g[i][q] = fma2(pre[i][q], suf[q], g[i][q]); suf[q] = mul2(suf[q], f[i][q]); }
#pragma unroll
            for (int q = 0; q < NP; ++q) g[0][q] = add2(g[0][q], suf[q]);     // prefix_0 = 1
        }
    }
    if constexpr (K >= 2) { if (n_cplx > 0) grp_rows_f2<K, NP, GRAD>(y, tabg, n_cplx, fe, g); }   // one of each conjugate pair, grouped
}

// sign flip by the literal's polarity bit (bit 31 of the packed literal): one LOP3 per value
__device__ __forceinline__ float flip_sign(float v, int32_t lit)
{
    return __int_as_float(__float_as_int(v) ^ (lit & LIT_NEG));
}
__device__ __forceinline__ double flip_sign(double v, int32_t lit)
{
    return __hiloint2double(__double2hiint(v) ^ (lit & LIT_NEG), __double2loint(v));
}

// One work item for this thread's V candidates; returns the item's partial objective in fe.
// Padding candidates (b >= B inside a live lane pair) are computed and scattered like live ones:
// G's padding columns are scratch here and are reset by the caller.
template <typename T, int K, int V, bool GRAD>
__device__ __forceinline__ void run_item_reg(const EvalParams<T> &p, const int32_t *__restrict__ s_lits,
                                             const T *__restrict__ s_tab, int n_real, int n_cplx, int nc, int wk,
                                             int64_t b, T (&fe)[V])
{
    const char *xb = reinterpret_cast<const char *>(p.x + b);
    char *gb = reinterpret_cast<char *>(p.G + (b - p.g_b0));
    const uint32_t x_ld = (uint32_t)(p.ldb * (int64_t)sizeof(T)), g_ld = (uint32_t)(p.g_ld * (int64_t)sizeof(T));
    const int Wk = p.Wk;
    for (int c = wk; c < nc; c += Wk) {
        const int32_t *L = s_lits + c * K;
        int32_t lit[K];
        T y[K][V], g[K][V];
#pragma unroll
        for (int i = 0; i < K; ++i) lit[i] = L[i];
#pragma unroll
        for (int i = 0; i < K; ++i) {
            VecIO<T, V>::load(reinterpret_cast<const T *>(xb + (uint64_t)(uint32_t)(lit[i] & LIT_VAR) * x_ld), y[i]);
#pragma unroll
            for (int v = 0; v < V; ++v) { y[i][v] = flip_sign(y[i][v], lit[i]); g[i][v] = T(0); }
        }
        eval_points_reg<T, K, V, GRAD>(y, s_tab, n_real, n_cplx, fe, g);
        if (GRAD) {
#pragma unroll
            for (int i = 0; i < K; ++i) {
                T gi[V];
#pragma unroll
                for (int v = 0; v < V; ++v) gi[v] = flip_sign(g[i][v], lit[i]);
                VecIO<T, V>::red(reinterpret_cast<T *>(gb + (uint64_t)(uint32_t)(lit[i] & LIT_VAR) * g_ld), gi);
            }
        }
    }
}

// The same for SHORT constraints, which are latency-bound on the gathers: the NEXT constraint's
// literals and row segments are requested before the current one is evaluated (software pipelining).
// Padding candidates (b >= B inside a live lane pair) are computed and scattered like live ones:
// G's padding columns are scratch here and are reset by the caller.
template <typename T, int K, int V, bool GRAD>
__device__ __forceinline__ void run_item_pf(const EvalParams<T> &p, const int32_t *__restrict__ s_lits,
                                             const T *__restrict__ s_tab, int n_real, int n_cplx, int nc, int wk,
                                             int64_t b, T (&fe)[V])
{
    const char *xb = reinterpret_cast<const char *>(p.x + b);
    char *gb = reinterpret_cast<char *>(p.G + (b - p.g_b0));
    const uint32_t x_ld = (uint32_t)(p.ldb * (int64_t)sizeof(T)), g_ld = (uint32_t)(p.g_ld * (int64_t)sizeof(T));
    const int Wk = p.Wk;
    int32_t lit_n[K];
    T y_n[K][V];
    auto fetch = [&](int c) {
        const int32_t *L = s_lits + c * K;
#pragma unroll
        for (int i = 0; i < K; ++i) lit_n[i] = L[i];
#pragma unroll
        for (int i = 0; i < K; ++i)
            VecIO<T, V>::load(reinterpret_cast<const T *>(xb + (uint64_t)(uint32_t)(lit_n[i] & LIT_VAR) * x_ld), y_n[i]);
    };
    if (wk < nc) fetch(wk);
    for (int c = wk; c < nc; c += Wk) {
        int32_t lit[K];
        T y[K][V], g[K][V];
#pragma unroll
        for (int i = 0; i < K; ++i) {
            lit[i] = lit_n[i];
#pragma unroll
            for (int v = 0; v < V; ++v) { y[i][v] = flip_sign(y_n[i][v], lit[i]); g[i][v] = T(0); }
        }
        if (c + Wk < nc) fetch(c + Wk);
        eval_points_reg<T, K, V, GRAD>(y, s_tab, n_real, n_cplx, fe, g);
        if (GRAD) {
#pragma unroll
            for (int i = 0; i < K; ++i) {
                T gi[V];
#pragma unroll
                for (int v = 0; v < V; ++v) gi[v] = flip_sign(g[i][v], lit[i]);
                VecIO<T, V>::red(reinterpret_cast<T *>(gb + (uint64_t)(uint32_t)(lit[i] & LIT_VAR) * g_ld), gi);
            }
        }
    }
}

// Stage the item's weight rows and literal list in shared memory (coalesced, once per CTA).
template <typename T>
__device__ __forceinline__ void stage_item(const EvalParams<T> &p, const Item &it, const SigDev &sg, T *s_tab,
                                           int32_t *s_lits)
{
    const int nrows8 = (sg.n_real + sg.n_cplx) * 8;
    for (int i = threadIdx.x; i < nrows8; i += blockDim.x) s_tab[i] = p.rows[(int64_t)sg.row_off * 8 + i];
    const int nl = (it.c_end - it.c_begin) * it.k;
    for (int i = threadIdx.x; i < nl; i += blockDim.x) s_lits[i] = __ldg(p.lits + it.lit_base + i);
}

// Sum the Wk warp groups' partial objectives in a fixed order and write Fpart[item][b].
template <typename T, int V>
__device__ __forceinline__ void store_item_F(const EvalParams<T> &p, T (*s_F)[32 * V], const T (&fe)[V], int warp,
                                             int lane, int wk, int64_t b, bool active)
{
    if (!p.Fpart) return;
#pragma unroll
    for (int v = 0; v < V; ++v) s_F[warp][lane * V + v] = fe[v];
    __syncthreads();
    if (wk == 0 && active) {
#pragma unroll
        for (int v = 0; v < V; ++v) {
            T s = T(0);
            for (int g = 0; g < p.Wk; ++g) s += s_F[warp + g * p.Wc][lane * V + v];
            if (b + v < p.B) p.Fpart[(int64_t)(p.frow_base + blockIdx.x) * p.ldb + b + v] = s;
        }
    }
}

// ---- packed-pair register kernel (fp32, NP pairs = 2 NP candidates per lane, FFMA2), length K --------
template <int NP> struct PairIO;
template <> struct PairIO<1> {
    static __device__ __forceinline__ void load(const char *p, f32x2 (&v)[1]) { v[0] = __ldg(reinterpret_cast<const f32x2 *>(p)); }
    static __device__ __forceinline__ void red(char *p, const f32x2 (&v)[1])
    {
        float a, b; upk(v[0], a, b);
        asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" ::"l"(p), "f"(a), "f"(b) : "memory");
    }
};
template <> struct PairIO<2> {
    static __device__ __forceinline__ void load(const char *p, f32x2 (&v)[2])
    {
        const ulonglong2 t = __ldg(reinterpret_cast<const ulonglong2 *>(p));
        v[0] = t.x; v[1] = t.y;
    }
    static __device__ __forceinline__ void red(char *p, const f32x2 (&v)[2])
    {
        float a, b, c, d; upk(v[0], a, b); upk(v[1], c, d);
        asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
    }
};

// PFD = how many constraints AHEAD of the one being evaluated the gathers are requested (register staging): 0 for the long
// bodies (k > 5: arithmetic hides the gathers), 1 for k = 4, 5, 2 for k <= 3 -- a k = 3 constraint is ~120 instructions per
// warp, too little to cover a loaded L2 round trip with one constraint in flight (ncu: the wait for the gathers was the
// top stall of cfg4's kernel, nearly all of it in the k = 3 body).
template <int K, int NP, int GRAD, int PFD, int UV>
__device__ __forceinline__ void run_item_f2(const EvalParams<float> &p, const int32_t *__restrict__ s_lits,
                                            const f32x2 *__restrict__ s_tab2, const float *__restrict__ s_tabg, int n_real,
                                            int n_cplx, int nc, int wk, int Wk, int64_t b, f32x2 (&fe)[NP])
{
    // wk / Wk: first constraint of this lane and the stride (lanes of a warp may walk different constraints, EvalParams::cs)
    const char *xb = reinterpret_cast<const char *>(p.x + b);
    char *gb = reinterpret_cast<char *>(p.G + (b - p.g_b0));
    const uint32_t x_ld = (uint32_t)(p.ldb * 4), g_ld = (uint32_t)(p.g_ld * 4);
    constexpr int NB = PFD > 1 ? PFD : 1;                             // staging buffers, used in turn
    int32_t lit_n[NB][K];
    f32x2 y_n[NB][K][NP];
    auto fetch = [&](int c, int32_t (&ln)[K], f32x2 (&yn)[K][NP]) {
        const int32_t *L = s_lits + c * K;
#pragma unroll
        for (int i = 0; i < K; ++i) ln[i] = L[i];
#pragma unroll
        for (int i = 0; i < K; ++i) PairIO<NP>::load(xb + (uint64_t)(uint32_t)(ln[i] & LIT_VAR) * x_ld, yn[i]);
    };
    // constraint c from its staging buffer; the buffer is then free for constraint c + PFD Wk
    auto one = [&](int c, int32_t (&ln)[K], f32x2 (&yn)[K][NP]) {
        if (PFD == 0) fetch(c, ln, yn);
        int32_t lit[K];
        f32x2 y[K][NP], g[K][NP];
#pragma unroll
        for (int i = 0; i < K; ++i) {
            lit[i] = ln[i];
            // y = s x as ONE packed multiply by (s, s), s = +-1 (exact: the same bits as flipping the two sign bits with two
            // LOP3s, -0.0 included, in half the issue slots)
            const f32x2 sf = bcf(__int_as_float(0x3f800000 | (lit[i] & LIT_NEG)));
#pragma unroll
            for (int q = 0; q < NP; ++q) { y[i][q] = mul2(yn[i][q], sf); g[i][q] = 0ull; }
        }
        if (PFD > 0 && c + PFD * Wk < nc) fetch(c + PFD * Wk, ln, yn);
        eval_points_f2<K, NP, GRAD, UV>(y, s_tab2, s_tabg, n_real, n_cplx, fe, g);
        if (GRAD) {
#pragma unroll
            for (int i = 0; i < K; ++i) {
                const f32x2 sf = bcf(__int_as_float(0x3f800000 | (lit[i] & LIT_NEG)));       // d/dx = s d/dy
                f32x2 gi[NP];
#pragma unroll
                for (int q = 0; q < NP; ++q) gi[q] = mul2(g[i][q], sf);
                PairIO<NP>::red(gb + (uint64_t)(uint32_t)(lit[i] & LIT_VAR) * g_ld, gi);
            }
        }
    };
#pragma unroll
    for (int u = 0; u < PFD; ++u)
        if (wk + u * Wk < nc) fetch(wk + u * Wk, lit_n[u], y_n[u]);
    for (int c = wk; c < nc; c += NB * Wk) {
#pragma unroll
        for (int u = 0; u < NB; ++u)
            if (u == 0 || c + u * Wk < nc) one(c + u * Wk, lit_n[u], y_n[u]);
    }
}

// ---- one launch for a RANGE of lengths [KLO, KHI]: the CTA's item picks its length-K body; all lengths share one grid
// (no per-length launch tails).  The bodies are INLINED into the kernel: as noinline functions (round 1, most of round 2)
// they could not keep the global-memory descriptor in uniform registers -- two R2UR before every gather and RED -- and
// spilled loop state around the call: cfg4 141 M -> 131 M warp instructions per launch, 266 -> 237 us ----
template <int K, int NP, int GRAD, bool CSPLIT>
__device__ __forceinline__ void item_body_f2(const EvalParams<float> &p, const int32_t *s_lits, const f32x2 *s_tab2,
                                          const float *s_tabg, float (*s_F)[64 * NP], int n_real, int n_cplx, int nc, int uv)
{
    constexpr int V = 2 * NP;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int wc = warp % p.Wc, wk = warp / p.Wc;
    // the warp's lanes take cs constraints at once (a narrow candidate tile still fills the warp: cfg4's tile of 64
    // candidates is 16 lanes x 4 candidates; the per-constraint instructions are issued once for both constraints)
    const int pcs = CSPLIT ? p.cs : 1;                                // (a compile-time 1 saves the registers of the general case)
    const int lpc = 32 / pcs, sub = lane / lpc, ll = lane % lpc;
    const int64_t b = p.b_begin + ((int64_t)blockIdx.y * p.Wc + wc) * (lpc * V) + ll * V;
    const bool active = b < p.b_end && b < p.B && !lane_skipped(p, b, V);   // this launch owns [b_begin, b_end)
    f32x2 fe2[NP];
#pragma unroll
    for (int q = 0; q < NP; ++q) fe2[q] = 0ull;
    if (active) {
        constexpr int PF = K <= 3 ? 2 : K <= 5 ? 1 : 0;
        const int c0 = wk * pcs + sub, cstep = p.Wk * pcs;
        if (uv == 1) run_item_f2<K, NP, GRAD, PF, 1>(p, s_lits, s_tab2, s_tabg, n_real, n_cplx, nc, c0, cstep, b, fe2);
        else if (uv == 2) run_item_f2<K, NP, GRAD, PF, 2>(p, s_lits, s_tab2, s_tabg, n_real, n_cplx, nc, c0, cstep, b, fe2);
        else run_item_f2<K, NP, GRAD, PF, 0>(p, s_lits, s_tab2, s_tabg, n_real, n_cplx, nc, c0, cstep, b, fe2);
    }
    if (!p.Fpart) return;
    // partial objectives: fixed-order sum over the Wk warp groups and the cs lane groups that hold the same candidates
    float fe[V];
#pragma unroll
    for (int q = 0; q < NP; ++q) upk(fe2[q], fe[2 * q], fe[2 * q + 1]);
#pragma unroll
    for (int v = 0; v < V; ++v) s_F[warp][lane * V + v] = fe[v];
    __syncthreads();
    if (wk == 0 && sub == 0 && active) {
#pragma unroll
        for (int v = 0; v < V; ++v) {
            float sacc = 0.f;
            for (int g = 0; g < p.Wk; ++g)
                for (int u = 0; u < pcs; ++u) sacc += s_F[warp + g * p.Wc][(u * lpc + ll) * V + v];
            if (b + v < p.B) p.Fpart[(int64_t)(p.frow_base + blockIdx.x) * p.ldb + b + v] = sacc;
        }
    }
}

template <int K, int KHI, int NP, int GRAD, bool CSPLIT>
struct SwitchF2 {
    static __device__ __forceinline__ void go(int k, const EvalParams<float> &p, const int32_t *s_lits, const f32x2 *s_tab2,
                                              const float *s_tabg, float (*s_F)[64 * NP], int n_real, int n_cplx, int nc, int uv)
    {
        if (k == K) item_body_f2<K, NP, GRAD, CSPLIT>(p, s_lits, s_tab2, s_tabg, s_F, n_real, n_cplx, nc, uv);
        else if (K < KHI) SwitchF2<(K < KHI ? K + 1 : K), KHI, NP, GRAD, CSPLIT>::go(k, p, s_lits, s_tab2, s_tabg, s_F, n_real, n_cplx, nc, uv);
    }
};

template <int KLO, int KHI, int NP, int GRAD, int MINB, bool CSPLIT>
__global__ void __launch_bounds__(CTA_THREADS, MINB) k_eval_f2m(const EvalParams<float> p)
{
    constexpr int H = (KHI + 1) / 2 + 1;
    __shared__ __align__(16) f32x2 s_tab2[(H + 2) * ROW2];
    __shared__ float s_tabg[H * ROW2G];
    __shared__ int32_t s_lits[LIT_CHUNK];
    __shared__ float s_F[CTA_WARPS][64 * NP];
    const Item it = p.items[blockIdx.x];
    const SigDev sg = p.sigs[it.sig];
    // the staged table (row order, folded weights: pack_rows_f2, built once per signature at create time)
    const int uv = sg.uv, n_unit = sg.n_unit, n_gen = sg.n_gen;
    for (int i = threadIdx.x; i < (n_unit + n_gen) * ROW2; i += blockDim.x) {
        const float v = __ldg(p.rows2 + (int64_t)sg.row2_off * ROW2 + i);
        s_tab2[i] = pk(v, v);
    }
    for (int i = threadIdx.x; i < n_gen * ROW2G; i += blockDim.x) s_tabg[i] = __ldg(p.rows2g + (int64_t)sg.row2g_off * ROW2G + i);
    const int nl = (it.c_end - it.c_begin) * it.k;
    for (int i = threadIdx.x; i < nl; i += blockDim.x) s_lits[i] = __ldg(p.lits + it.lit_base + i);
    __syncthreads();
    SwitchF2<KLO, KHI, NP, GRAD, CSPLIT>::go(it.k, p, s_lits, s_tab2, s_tabg, s_F, n_unit, n_gen, it.c_end - it.c_begin, uv);
}

// one body per length, fp64 k <= 8 (everything longer, and fp32 beyond k = 8, runs the lane-split kernels of afsat_split.cuh)
template <typename T, int K, int V, bool GRAD>
__device__ __forceinline__ void item_body_k(const EvalParams<T> &p, const int32_t *s_lits, const T *s_tab, T (*s_F)[32 * V],
                                         int n_real, int n_cplx, int nc)
{
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int wc = warp % p.Wc, wk = warp / p.Wc;
    const int64_t b = p.b_begin + ((int64_t)blockIdx.y * p.Wc + wc) * (32 * V) + lane * V;
    const bool active = b < p.b_end && b < p.B && !lane_skipped(p, b, V);   // this launch owns [b_begin, b_end)
    T fe[V];
#pragma unroll
    for (int v = 0; v < V; ++v) fe[v] = T(0);
    if (active) {
        if (K <= 5) run_item_pf<T, K, V, GRAD>(p, s_lits, s_tab, n_real, n_cplx, nc, wk, b, fe);
        else run_item_reg<T, K, V, GRAD>(p, s_lits, s_tab, n_real, n_cplx, nc, wk, b, fe);
    }
    store_item_F<T, V>(p, s_F, fe, warp, lane, wk, b, active);
}

template <typename T, int K, int KHI, int V, bool GRAD>
struct SwitchK {
    static __device__ __forceinline__ void go(int k, const EvalParams<T> &p, const int32_t *s_lits, const T *s_tab,
                                              T (*s_F)[32 * V], int n_real, int n_cplx, int nc)
    {
        if (k == K) item_body_k<T, K, V, GRAD>(p, s_lits, s_tab, s_F, n_real, n_cplx, nc);
        else if (K < KHI) SwitchK<T, (K < KHI ? K + 1 : K), KHI, V, GRAD>::go(k, p, s_lits, s_tab, s_F, n_real, n_cplx, nc);
    }
};

template <typename T, int KLO, int KHI, int V, bool GRAD, int MINB>
__global__ void __launch_bounds__(CTA_THREADS, MINB) k_eval_km(const EvalParams<T> p)
{
    __shared__ __align__(16) T s_tab[((KHI + 1) / 2 + 1) * 8];
    __shared__ int32_t s_lits[LIT_CHUNK];
    __shared__ T s_F[CTA_WARPS][32 * V];
    const Item it = p.items[blockIdx.x];
    const SigDev sg = p.sigs[it.sig];
    stage_item(p, it, sg, s_tab, s_lits);
    __syncthreads();
    SwitchK<T, KLO, KHI, V, GRAD>::go(it.k, p, s_lits, s_tab, s_F, sg.n_real, sg.n_cplx, it.c_end - it.c_begin);
}

// length classes (afsat.cu class_of): fp32  k <= 5: k_eval_f2m, four candidates per lane | 6..8: k_eval_f2m, two per lane |
// 9..20: packed lane-split kernel | 21..64: scalar lane-split kernel;  fp64  k <= 8: k_eval_km | 9..20, 21..64: lane-split
#define AFSAT_S_KMAX 5
#define AFSAT_A_KMAX 8
#define AFSAT_B_KMAX 20

}  // namespace afsat
