// afsat.cu -- C ABI (include/afsat.h) of the B200-native AFSAT hot path: context construction
// (validation, bucketing by signature and length, table upload) and the launch sequences of
// afsat_eval_grad / afsat_check / afsat_step.  All arithmetic of the path runs in the kernels of
// afsat_kernels.cuh; the host tables come from precompute.cpp.  No CPU fallback exists.
#include <cuda_runtime.h>
#include <algorithm>
#include <map>
#include <new>
#include <string>
#include <tuple>
#include <vector>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "afsat_internal.h"
#include "afsat_kernels.cuh"
#include "afsat_split.cuh"

using namespace afsat;

// tuning knobs of the k <= 8 fp32 register kernel: candidates per lane and
// the occupancy the register allocator is held to
#ifndef AFSAT_A_V
#define AFSAT_A_V 2
#endif
#ifndef AFSAT_A_MINB
#define AFSAT_A_MINB 2
#endif

namespace {

thread_local std::string g_create_error;

// length classes: register kernels for k in [1,8] and [9,16] (one launch each, one separately compiled
// body per length), shared-memory kernel for [17,64]
// fp32 only: the shortest constraints (k <= AFSAT_S_KMAX) run FOUR candidates per lane (two packed pairs): their
// launches are issue-bound on per-constraint overhead (literal and table loads, addresses, sign masks), which
// a lane then pays once per four candidates; their bodies are small enough for it at 128 registers
#ifndef AFSAT_S_KMAX
#define AFSAT_S_KMAX 5
#endif
#if defined(AFSAT_NO_FFMA2) || AFSAT_A_V < 2
#undef AFSAT_S_KMAX
#define AFSAT_S_KMAX 0
#endif
// fp32: the scalar register kernel (one candidate per lane, every intermediate in registers, the compiler
// spilling what does not fit) up to this length; it beats the shared-memory-staged kernel at every length
#ifndef AFSAT_B_KMAX64
#define AFSAT_B_KMAX64 20
#endif
enum { CLS_S = 0, CLS_A = 1, CLS_B = 2, CLS_LONG = 3, N_CLS = 4 };
inline int class_of(int k, int dtype)
{
    return (dtype == 32 && k <= AFSAT_S_KMAX) ? CLS_S : k <= 8 ? CLS_A : k <= (dtype == 32 ? AFSAT_B_KMAX32 : AFSAT_B_KMAX64) ? CLS_B : CLS_LONG;
}

struct ClassGeom {              // how one length class maps candidates onto a CTA
    int V = 1;                  // candidates per lane
    int cw = 32;                // candidates per warp (32 V; 32 / NS in the lane-split kernel)
    int warps = CTA_WARPS;      // warps per CTA
    int Wc = 1, Wk = CTA_WARPS; // candidate sub-tiles x constraint groups
    size_t smem = 0;            // dynamic shared memory (long kernel only)
};

}  // namespace

struct afsat_ctx {
    int32_t n = 0, m = 0, B = 0, dtype = 32, device = 0, sm_count = 148;
    int64_t ldb = 0, nnz = 0, tile_w = 0;
    uint32_t flags = 0;
    size_t esz = 4;
    // device tables
    int32_t *d_lits = nullptr;
    SigDev *d_sigs = nullptr;
    void *d_rows = nullptr;
    float *d_rows2 = nullptr;                      // staged tables of the packed fp32 kernel
    int8_t *d_fixed = nullptr;
    Item *d_items = nullptr;
    int32_t n_items = 0, cls_begin[N_CLS + 1] = {0};
    ClassGeom geom[N_CLS];
    int32_t kmax_long = 0;
    int32_t n_sigs = 0, n_buckets = 0;
    int64_t fp_instr_per_candidate = 0;
    // workspace
    void *d_G = nullptr, *d_Fpart = nullptr;      // G scratch [n][tile_w]; Fpart [n_items][ldb]
    uint32_t *d_bits = nullptr;                    // sign bits [n][ldb/32]
    int32_t *d_satacc = nullptr, *d_any = nullptr;
    // buffers of afsat_step_host (lazy)
    void *dh_x = nullptr, *dh_F = nullptr;
    int32_t *dh_sat = nullptr, *dh_first = nullptr;
    uint8_t *dh_sol = nullptr;
    // workspace of afsat_step_ls (lazy): full gradient, trial X', reduction partials, per-candidate state
    void *ls_G = nullptr, *ls_xt = nullptr, *ls_F0 = nullptr, *ls_F1 = nullptr;
    double *ls_Dpart = nullptr, *ls_eta = nullptr;
    uint8_t *ls_state = nullptr;
    const uint8_t *cur_skip = nullptr;             // candidate mask of the evaluation launches (line-search trials)
    cudaStream_t own_stream = nullptr;
    cudaStream_t side_stream[N_CLS - 1] = {};                       // concurrent launches of the length classes
    cudaEvent_t ev_fork = nullptr, ev_join[N_CLS - 1] = {};
    size_t ws_bytes = 0;
    int64_t launches = 0;
    // afsat_set_profiling: event pairs around the evaluation-kernel launches
    bool profiling = false;
    std::vector<std::pair<cudaEvent_t, cudaEvent_t>> prof_events;
    double prof_ns = 0.0;
    int64_t prof_launches = 0;
    std::string err;
};

namespace {

int fail(afsat_ctx *c, int code, const std::string &msg)
{
    if (c) c->err = msg; else g_create_error = msg;
    return code;
}

#define CU(call)                                                                               \
    do {                                                                                       \
        cudaError_t e_ = (call);                                                               \
        if (e_ != cudaSuccess)                                                                 \
            return fail(ctx, AFSAT_E_CUDA, std::string(#call) + ": " + cudaGetErrorString(e_)); \
    } while (0)

template <typename U>
int dev_alloc(afsat_ctx *ctx, U **p, size_t count, bool zero = false)
{
    size_t bytes = std::max<size_t>(count, 1) * sizeof(U);
    CU(cudaMalloc((void **)p, bytes));
    ctx->ws_bytes += bytes;
    if (zero) CU(cudaMemset(*p, 0, bytes));
    return AFSAT_OK;
}

template <typename U>
int upload(afsat_ctx *ctx, U **p, const std::vector<U> &h)
{
    int rc = dev_alloc(ctx, p, h.size());
    if (rc) return rc;
    if (!h.empty()) CU(cudaMemcpy(*p, h.data(), h.size() * sizeof(U), cudaMemcpyHostToDevice));
    return AFSAT_OK;
}

// model count of FP instructions for one (constraint, candidate): DESIGN.md cost model
inline int64_t cost_of(int k, int n_real, int n_cplx) { return (int64_t)k * (12 * n_cplx + 4 * n_real) + 2 * n_cplx + n_real; }

inline int pow2_floor(int64_t v) { int p = 1; while ((int64_t)p * 2 <= v) p *= 2; return p; }

// brackets one evaluation-kernel launch with events when profiling is on
struct ProfScope {
    afsat_ctx *c; cudaStream_t st; cudaEvent_t e0 = nullptr, e1 = nullptr;
    ProfScope(afsat_ctx *c_, cudaStream_t st_) : c(c_), st(st_)
    {
        if (!c->profiling) return;
        if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) { e0 = e1 = nullptr; return; }
        cudaEventRecord(e0, st);
    }
    ~ProfScope()
    {
        if (!e0) return;
        cudaEventRecord(e1, st);
        c->prof_events.emplace_back(e0, e1);
    }
};

void prof_drain(afsat_ctx *c, bool keep)
{
    for (auto &pr : c->prof_events) {
        if (keep && cudaEventSynchronize(pr.second) == cudaSuccess) {
            float ms = 0.f;
            if (cudaEventElapsedTime(&ms, pr.first, pr.second) == cudaSuccess) { c->prof_ns += (double)ms * 1e6; ++c->prof_launches; }
        }
        cudaEventDestroy(pr.first); cudaEventDestroy(pr.second);
    }
    c->prof_events.clear();
}

// k <= 8: fp32 with >= 2 candidates per lane runs the packed FFMA2 kernel, everything else the scalar one
template <typename T, int VA, int MB>
void (*pick_a(bool grad))(EvalParams<T>)
{
    using Fn = void (*)(EvalParams<T>);
#ifndef AFSAT_NO_FFMA2
    if constexpr (sizeof(T) == 4 && VA >= 2) return grad ? (Fn)k_eval_f2m<1, 8, VA / 2, true, MB> : (Fn)k_eval_f2m<1, 8, VA / 2, false, MB>;
    else
#endif
        return grad ? (Fn)k_eval_km<T, 1, 8, VA, true, MB> : (Fn)k_eval_km<T, 1, 8, VA, false, MB>;
}

// k <= AFSAT_S_KMAX, fp32: the packed kernel with two pairs (four candidates) per lane
template <typename T, int MB>
void (*pick_s(bool grad))(EvalParams<T>)
{
    using Fn = void (*)(EvalParams<T>);
#if AFSAT_S_KMAX > 0
    if constexpr (sizeof(T) == 4) return grad ? (Fn)k_eval_f2m<1, AFSAT_S_KMAX, 2, true, MB> : (Fn)k_eval_f2m<1, AFSAT_S_KMAX, 2, false, MB>;
    else
#endif
        return nullptr;                                                // class S is empty for this dtype / build
}

template <typename T>
void (*pick_b(bool grad))(EvalParams<T>)
{
    using Fn = void (*)(EvalParams<T>);
    constexpr int KHI = sizeof(T) == 4 ? AFSAT_B_KMAX32 : AFSAT_B_KMAX64;
#if AFSAT_M32_PACKED
    if constexpr (sizeof(T) == 4)                                      // fp32: the packed lane-split kernel
        return grad ? (Fn)k_eval_split<float, 9, AFSAT_B_KMAX32, 2, 2, true, AFSAT_M32_THREADS, 1>
                    : (Fn)k_eval_split<float, 9, AFSAT_B_KMAX32, 2, 2, false, AFSAT_M32_THREADS, 1>;
    else
#endif
    return grad ? (Fn)k_eval_km<T, 9, KHI, 1, true, AFSAT_B_MINB> : (Fn)k_eval_km<T, 9, KHI, 1, false, AFSAT_B_MINB>;
}

// k > 16: KMAX is the unroll bound of the register-blocked kernels; fp32 runs the packed two-candidate form
inline int long_kmax(int kmax_long) { return kmax_long <= 32 ? 32 : kmax_long <= 40 ? 40 : kmax_long <= 48 ? 48 : kmax_long <= 56 ? 56 : 64; }
template <typename T>
void (*pick_long(int km, bool grad))(EvalParams<T>)
{
    using Fn = void (*)(EvalParams<T>);
    if constexpr (sizeof(T) == 4) {                                    // fp32: the lane-split register kernel
        return grad ? (Fn)k_eval_split<float, AFSAT_L32_KMIN, AFSAT_MAX_LEN, AFSAT_L32_NS, 1, true, AFSAT_L32_THREADS, AFSAT_L32_MINB>
                    : (Fn)k_eval_split<float, AFSAT_L32_KMIN, AFSAT_MAX_LEN, AFSAT_L32_NS, 1, false, AFSAT_L32_THREADS, AFSAT_L32_MINB>;
    } else {
#if AFSAT_L64_SPLIT
        return grad ? (Fn)k_eval_split<double, AFSAT_L64_KMIN, AFSAT_MAX_LEN, 4, 1, true, AFSAT_L64_THREADS, 1>
                    : (Fn)k_eval_split<double, AFSAT_L64_KMIN, AFSAT_MAX_LEN, 4, 1, false, AFSAT_L64_THREADS, 1>;
#endif
#define AFSAT_LONG_CASE(KM_)                                                                                  \
    case KM_:                                                                                                 \
        return grad ? (Fn)k_eval_blk<T, KM_, true> : (Fn)k_eval_blk<T, KM_, false>;
    switch (km) {
        AFSAT_LONG_CASE(32) AFSAT_LONG_CASE(40) AFSAT_LONG_CASE(48) AFSAT_LONG_CASE(56)
    default:
        AFSAT_LONG_CASE(64)
    }
#undef AFSAT_LONG_CASE
    }
}

// ---- launch of the evaluation kernels (a1-a5) for the candidate tile [b_begin, b_begin + width) ----
template <typename T>
int launch_eval(afsat_ctx *ctx, const T *x, T *G, int64_t g_ld, int64_t g_b0, T *Fpart, int64_t b_begin, int64_t width,
                cudaStream_t st)
{
    EvalParams<T> p;
    p.x = x; p.G = G; p.g_ld = g_ld; p.g_b0 = g_b0; p.Fpart = Fpart;
    p.lits = ctx->d_lits; p.sigs = ctx->d_sigs; p.rows = (const T *)ctx->d_rows; p.rows2 = ctx->d_rows2;
    p.skip = ctx->cur_skip;
    p.B = ctx->B; p.ldb = ctx->ldb; p.b_begin = b_begin; p.b_end = std::min<int64_t>(b_begin + width, ctx->ldb);
    const bool grad = G != nullptr;
    constexpr int VA = sizeof(T) == 4 ? AFSAT_A_V : 1;
    // The length classes are independent (they only share the RED target), so their launches run
    // CONCURRENTLY: class 0 on the caller's stream, the others on forked side streams that join back.
    int n_active = 0;
    for (int cls = 0; cls < N_CLS; ++cls) n_active += ctx->cls_begin[cls + 1] > ctx->cls_begin[cls];
    ProfScope prof(ctx, st);                                          // brackets the whole launch set
    const bool fork = n_active > 1;
    if (fork) CU(cudaEventRecord(ctx->ev_fork, st));
    int side = 0;
    cudaStream_t user_st = st;
    for (int cls = 0; cls < N_CLS; ++cls) {
        const int nit = ctx->cls_begin[cls + 1] - ctx->cls_begin[cls];
        if (nit == 0) continue;
        st = user_st;
        int my_side = -1;
        if (fork && side < N_CLS - 1 && cls != 0 && ctx->cls_begin[cls] != 0) {   // not the first active class
            my_side = side++;
            st = ctx->side_stream[my_side];
            CU(cudaStreamWaitEvent(st, ctx->ev_fork, 0));
        }
        const ClassGeom &g = ctx->geom[cls];
        p.items = ctx->d_items + ctx->cls_begin[cls];
        p.frow_base = ctx->cls_begin[cls];
        p.Wc = g.Wc; p.Wk = g.Wk;
        const int64_t per_cta = (int64_t)g.cw * g.Wc;
        dim3 block(32 * g.warps), grid(nit, (unsigned)((width + per_cta - 1) / per_cta));
        if (cls != CLS_LONG) {
            using Fn = void (*)(EvalParams<T>);
            constexpr int MB = sizeof(T) == 4 ? AFSAT_A_MINB : 1;
            Fn fn = cls == CLS_S ? pick_s<T, MB>(grad)
                  : cls == CLS_A ? pick_a<T, VA, MB>(grad)
                                 : pick_b<T>(grad);
            fn<<<grid, block, 0, st>>>(p);
        } else {
            using Fn = void (*)(EvalParams<T>);
            Fn fn = pick_long<T>(long_kmax(ctx->kmax_long), grad);
            if (g.smem) CU(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)g.smem));
            fn<<<grid, block, g.smem, st>>>(p);
        }
        ++ctx->launches;
        CU(cudaPeekAtLastError());
        if (my_side >= 0) {
            CU(cudaEventRecord(ctx->ev_join[my_side], st));
            CU(cudaStreamWaitEvent(user_st, ctx->ev_join[my_side], 0));
        }
    }
    return AFSAT_OK;
}

// a8 on the words [w_begin, w_end) of the sign-bit array
int launch_check_bits(afsat_ctx *ctx, int64_t w_begin, int64_t w_end, cudaStream_t st)
{
    if (ctx->n_items == 0 || w_end <= w_begin) return AFSAT_OK;
    CheckParams p;
    p.bits = ctx->d_bits; p.ldw = ctx->ldb / 32; p.lits = ctx->d_lits; p.sigs = ctx->d_sigs; p.items = ctx->d_items;
    p.satacc = ctx->d_satacc; p.B = ctx->B; p.w_begin = (int32_t)w_begin; p.w_end = (int32_t)w_end;
    const int64_t nw = w_end - w_begin;
    p.wpb = std::min(32, pow2_floor(nw));
    if (p.wpb < nw && p.wpb < 32) p.wpb *= 2;                         // cover a ragged word count in one CTA row
    p.wpb = std::min(p.wpb, 32);
    p.n_items = ctx->n_items;
    const unsigned gy = (unsigned)((nw + p.wpb - 1) / p.wpb);
    dim3 grid((unsigned)std::max<int64_t>(1, std::min<int64_t>(ctx->n_items, (int64_t)ctx->sm_count * 4 / gy)), gy);
    k_check_bits<<<grid, CTA_THREADS, 0, st>>>(p);
    ++ctx->launches;
    CU(cudaPeekAtLastError());
    return AFSAT_OK;
}

template <typename T>
int launch_pack(afsat_ctx *ctx, const T *x, cudaStream_t st)
{
    const unsigned gx = (unsigned)((ctx->ldb + CTA_THREADS - 1) / CTA_THREADS);
    const unsigned gy = (unsigned)std::min<int64_t>(ctx->n, std::max<int64_t>(1, (int64_t)ctx->sm_count * 8 / gx));
    k_pack_signs<T><<<dim3(gx, gy), CTA_THREADS, 0, st>>>(x, ctx->d_bits, ctx->n, ctx->B, ctx->ldb);
    ++ctx->launches;
    CU(cudaPeekAtLastError());
    return AFSAT_OK;
}

template <typename T>
int reduce_F(afsat_ctx *ctx, T *F, cudaStream_t st)
{
    k_reduce_F<T><<<(ctx->B + 127) / 128, 128, 0, st>>>((const T *)ctx->d_Fpart, ctx->n_items, ctx->ldb, ctx->B, F, ctx->cur_skip);
    ++ctx->launches;
    CU(cudaPeekAtLastError());
    return AFSAT_OK;
}

template <typename T>
int eval_grad_t(afsat_ctx *ctx, const T *x, T *F, T *G, cudaStream_t st)
{
    if (G) CU(cudaMemsetAsync(G, 0, (size_t)ctx->n * ctx->ldb * sizeof(T), st));
    for (int64_t b0 = 0; b0 < ctx->B; b0 += ctx->tile_w) {            // candidate tiles keep X/G tiles L2-resident
        const int64_t w = std::min<int64_t>(ctx->tile_w, ctx->ldb - b0);
        int rc = launch_eval<T>(ctx, x, G, ctx->ldb, 0, F ? (T *)ctx->d_Fpart : nullptr, b0, w, st);
        if (rc) return rc;
    }
    if (G && ctx->B < ctx->ldb && (ctx->B & 3)) {                     // a lane's candidates straddle B: clear the spill
        k_zero_pad<T><<<std::min(1024, ctx->n), 128, 0, st>>>(G, ctx->n, ctx->B, ctx->ldb);
        ++ctx->launches;
        CU(cudaPeekAtLastError());
    }
    if (F) return reduce_F<T>(ctx, F, st);
    return AFSAT_OK;
}

template <typename T>
int step_t(afsat_ctx *ctx, T *x, double eta, int n_steps, int step_base, int resume, T *F, int32_t *sat,
           uint8_t *sol, int32_t *first, int32_t *h_any_dev, cudaStream_t st)
{
    const int B = ctx->B, tb = 128, gb = (B + tb - 1) / tb;
    if (!resume) {
        k_reset_state<<<gb, tb, 0, st>>>(B, sol, first);
        ++ctx->launches;
    }
    CU(cudaMemsetAsync(ctx->d_any, 0, 2 * sizeof(int32_t), st));
    const int64_t tw = ctx->tile_w;
    for (int t = 1; t <= n_steps; ++t) {
        for (int64_t b0 = 0; b0 < B; b0 += tw) {
            const int64_t w = std::min<int64_t>(tw, ctx->ldb - b0);
            // a1-a5: gradient at X(t-1) into the (zeroed) tile scratch
            int rc = launch_eval<T>(ctx, x, (T *)ctx->d_G, tw, b0, nullptr, b0, w, st);
            if (rc) return rc;
            // a6, a7, a9: X(t) = clamp(X(t-1) - eta G) on free variables of unsolved candidates, sign bits, G reset
            const int cols = (int)std::min<int64_t>(CTA_THREADS, w);                 // w is a multiple of 32
            const int ucols = CTA_THREADS % cols == 0 ? cols : 32;
            const unsigned gx = (unsigned)((w + ucols - 1) / ucols);
            const int rpp = CTA_THREADS / ucols;
            const unsigned gy = (unsigned)std::max<int64_t>(1, std::min<int64_t>((ctx->n + rpp * UPD_UNROLL - 1) / (rpp * UPD_UNROLL),
                                                                                   (int64_t)ctx->sm_count * 8 / gx));
            k_update<T><<<dim3(gx, gy), CTA_THREADS, 0, st>>>(x, (T *)ctx->d_G, tw, b0, ctx->d_fixed, sol, ctx->d_bits, (T)eta,
                                                              ctx->n, B, ctx->ldb, b0, b0 + w, ucols);
            ++ctx->launches;
            CU(cudaPeekAtLastError());
        }
        // a8: exact count on X(t), ONE launch over the whole batch: every constraint reads the full
        // [ldb/32]-word bit rows of its variables (coalesced), 1 bit per literal and candidate
        {
            int rc = launch_check_bits(ctx, 0, ctx->ldb / 32, st);
            if (rc) return rc;
        }
        k_flags<<<gb, tb, 0, st>>>(ctx->d_satacc, B, ctx->m, 1, step_base + t, sat, sol, first, ctx->d_any, h_any_dev);
        ++ctx->launches;
        CU(cudaPeekAtLastError());
    }
    if (n_steps == 0) {                                               // no step: count on X as it is, mark nothing
        int rc = launch_pack<T>(ctx, x, st);
        if (!rc) rc = launch_check_bits(ctx, 0, ctx->ldb / 32, st);
        if (rc) return rc;
        k_flags<<<gb, tb, 0, st>>>(ctx->d_satacc, B, ctx->m, 0, step_base, sat, sol, first, ctx->d_any, h_any_dev);
        ++ctx->launches;
        CU(cudaPeekAtLastError());
    }
    if (F) {                                                          // objective at the final X
        for (int64_t b0 = 0; b0 < B; b0 += tw) {
            int rc = launch_eval<T>(ctx, x, nullptr, 0, 0, (T *)ctx->d_Fpart, b0, std::min<int64_t>(tw, ctx->ldb - b0), st);
            if (rc) return rc;
        }
        return reduce_F<T>(ctx, F, st);
    }
    return AFSAT_OK;
}

// Alg. 1 with the per-candidate backtracking line search of afsat_step_ls (include/afsat.h)
template <typename T>
int step_ls_t(afsat_ctx *ctx, T *x, double s_max, double beta, double c1, double delta, int max_trials, int n_steps,
              int step_base, int resume, T *F, void *eta_out, int32_t *sat, uint8_t *sol, int32_t *first, uint8_t *conv,
              int32_t *h_any_dev, cudaStream_t st)
{
    const int B = ctx->B, tb = 128, gb = (B + tb - 1) / tb;
    const int64_t ldb = ctx->ldb;
    const size_t nb = (size_t)ctx->n * ldb;
    if (!ctx->ls_G) {
        int rc;
        char *pg = nullptr, *px = nullptr, *p0 = nullptr, *p1 = nullptr;
        if ((rc = dev_alloc(ctx, &pg, nb * sizeof(T)))) return rc;
        ctx->ls_G = pg;
        if ((rc = dev_alloc(ctx, &px, nb * sizeof(T)))) return rc;
        ctx->ls_xt = px;
        if ((rc = dev_alloc(ctx, &p0, (size_t)ldb * sizeof(T), true))) return rc;
        ctx->ls_F0 = p0;
        if ((rc = dev_alloc(ctx, &p1, (size_t)ldb * sizeof(T), true))) return rc;
        ctx->ls_F1 = p1;
        if ((rc = dev_alloc(ctx, &ctx->ls_Dpart, (size_t)LS_CHUNKS * ldb, true))) return rc;
        if ((rc = dev_alloc(ctx, &ctx->ls_eta, (size_t)ldb, true))) return rc;
        if ((rc = dev_alloc(ctx, &ctx->ls_state, (size_t)ldb, true))) return rc;
    }
    T *G = (T *)ctx->ls_G, *xt = (T *)ctx->ls_xt, *F0 = (T *)ctx->ls_F0, *F1 = (T *)ctx->ls_F1;
    if (!resume) {
        k_reset_state<<<gb, tb, 0, st>>>(B, sol, first);
        ++ctx->launches;
        CU(cudaMemsetAsync(conv, 0, (size_t)B, st));
    }
    CU(cudaMemsetAsync(ctx->d_any, 0, 2 * sizeof(int32_t), st));
    const unsigned gl = (unsigned)((ldb + CTA_THREADS - 1) / CTA_THREADS);
    const unsigned gyc = (unsigned)std::min<int64_t>(ctx->n, std::max<int64_t>(1, (int64_t)ctx->sm_count * 8 / gl));
    if (n_steps == 0) {                                               // no step: F, counts on X as it is
        k_ls_begin<<<gl, CTA_THREADS, 0, st>>>(B, ldb, sol, conv, ctx->ls_state, s_max, ctx->ls_eta);
        ++ctx->launches;
        int rc = eval_grad_t<T>(ctx, x, F0, (T *)nullptr, st);
        if (!rc) rc = launch_pack<T>(ctx, x, st);
        if (!rc) rc = launch_check_bits(ctx, 0, ldb / 32, st);
        if (rc) return rc;
        k_flags<<<gb, tb, 0, st>>>(ctx->d_satacc, B, ctx->m, 0, step_base, sat, sol, first, ctx->d_any, h_any_dev);
        ++ctx->launches;
    }
    for (int t = 1; t <= n_steps; ++t) {
        k_ls_begin<<<gl, CTA_THREADS, 0, st>>>(B, ldb, sol, conv, ctx->ls_state, s_max, ctx->ls_eta);
        ++ctx->launches;
        // a1-a5 at X(t-1): objective and full gradient (frozen candidates are skipped)
        ctx->cur_skip = ctx->ls_state;
        int rc = eval_grad_t<T>(ctx, x, F0, G, st);
        ctx->cur_skip = nullptr;
        if (rc) return rc;
        for (int j = 0; j < max_trials; ++j) {
            k_ls_trial<T><<<dim3(gl, LS_CHUNKS), CTA_THREADS, 0, st>>>(x, G, xt, ctx->d_fixed, ctx->ls_state, ctx->ls_eta,
                                                                        ctx->ls_Dpart, ctx->n, ldb, j == 0);
            ++ctx->launches;
            CU(cudaPeekAtLastError());
            ctx->cur_skip = ctx->ls_state;                            // objective only, candidates still searching
            rc = eval_grad_t<T>(ctx, xt, F1, (T *)nullptr, st);
            ctx->cur_skip = nullptr;
            if (rc) return rc;
            k_ls_decide<T><<<gb, tb, 0, st>>>(B, ldb, F0, F1, ctx->ls_Dpart, ctx->ls_state, ctx->ls_eta, conv, c1, beta, delta);
            ++ctx->launches;
            CU(cudaPeekAtLastError());
        }
        k_ls_commit<T><<<dim3(gl, gyc), CTA_THREADS, 0, st>>>(x, xt, ctx->ls_state, ctx->d_bits, ctx->n, B, ldb);
        ++ctx->launches;
        CU(cudaPeekAtLastError());
        rc = launch_check_bits(ctx, 0, ldb / 32, st);
        if (rc) return rc;
        k_flags<<<gb, tb, 0, st>>>(ctx->d_satacc, B, ctx->m, 1, step_base + t, sat, sol, first, ctx->d_any, h_any_dev);
        ++ctx->launches;
        CU(cudaPeekAtLastError());
    }
    if (eta_out) {
        k_ls_report<T><<<gb, tb, 0, st>>>(B, ctx->ls_eta, (T *)eta_out);
        ++ctx->launches;
        CU(cudaPeekAtLastError());
    }
    if (F && n_steps > 0) return eval_grad_t<T>(ctx, x, F, (T *)nullptr, st);   // objective at the final X, every candidate
    if (F) CU(cudaMemcpyAsync(F, F0, (size_t)B * sizeof(T), cudaMemcpyDeviceToDevice, st));
    return AFSAT_OK;
}

int set_device(afsat_ctx *ctx)
{
    CU(cudaSetDevice(ctx->device));
    return AFSAT_OK;
}

}  // namespace

// ============================================================================================
extern "C" {

const char *afsat_version(void) { return "afsat-b200 0.1 (sm_100a)"; }

const char *afsat_last_error(const afsat_ctx *ctx) { return ctx ? ctx->err.c_str() : g_create_error.c_str(); }

int afsat_host_tables(int32_t type, int32_t k, int32_t param, uint32_t flags, double *table, int32_t *n_real)
{
    if (!table) return AFSAT_E_INVALID;
    AfsatSigHost s;
    int rc = afsat_sig_build(type, k, param, flags, &s);
    if (rc) return rc;
    const int rows = s.n_real + s.n_cplx;
    memcpy(table, s.rows, sizeof(double) * 8 * rows);
    if (n_real) *n_real = s.n_real;
    return rows;
}

int afsat_create(afsat_ctx **out, int32_t n_vars, int32_t n_cons, const int64_t *row_ptr, const int32_t *lit_var,
                 const int8_t *lit_sign, const uint8_t *type, const int32_t *param, const int8_t *fixed,
                 int32_t batch, int64_t ldb, int32_t dtype, int32_t device, uint32_t flags)
{
    afsat_ctx *ctx = nullptr;   // errors before allocation go to the thread-local message
    if (!out) return fail(ctx, AFSAT_E_INVALID, "out is NULL");
    *out = nullptr;
    if (n_vars < 1 || n_vars > LIT_VAR) return fail(ctx, AFSAT_E_INVALID, "n_vars out of range");
    if (n_cons < 0) return fail(ctx, AFSAT_E_INVALID, "n_cons < 0");
    if (!row_ptr || (n_cons > 0 && (!type || !param))) return fail(ctx, AFSAT_E_INVALID, "NULL constraint arrays");
    if (batch < 1) return fail(ctx, AFSAT_E_INVALID, "batch must be >= 1");
    if (ldb < batch || ldb % 32 != 0) return fail(ctx, AFSAT_E_INVALID, "ldb must be >= batch and a multiple of 32");
    if (dtype != 32 && dtype != 64) return fail(ctx, AFSAT_E_INVALID, "dtype must be 32 or 64");
    if (flags & ~(uint32_t)AFSAT_FLAG_ROBUST) return fail(ctx, AFSAT_E_INVALID, "unknown flags");
    if (row_ptr[0] != 0) return fail(ctx, AFSAT_E_INVALID, "row_ptr[0] != 0");
    const int64_t nnz = row_ptr[n_cons];
    if (nnz > 0 && (!lit_var || !lit_sign)) return fail(ctx, AFSAT_E_INVALID, "NULL literal arrays");
    if (fixed)
        for (int32_t v = 0; v < n_vars; ++v)
            if (fixed[v] < -1 || fixed[v] > 1) return fail(ctx, AFSAT_E_SIGN, "fixed[] must be -1, 0 or +1");

    // ---- validate constraints, assign signatures -------------------------------------------
    std::map<std::tuple<int, int, int>, int> sig_id;            // (k, type, param) -> id, ordered by k
    std::vector<int32_t> csig(n_cons);
    std::vector<int32_t> scratch;
    for (int32_t c = 0; c < n_cons; ++c) {
        const int64_t lo = row_ptr[c], hi = row_ptr[c + 1];
        const int64_t k = hi - lo;
        char buf[160];
        if (k < 1 || k > AFSAT_MAX_LEN) {
            snprintf(buf, sizeof buf, "constraint %d has length %lld (allowed 1..%d)", c, (long long)k, AFSAT_MAX_LEN);
            return fail(ctx, AFSAT_E_LENGTH, buf);
        }
        if (type[c] > AFSAT_NAE) { snprintf(buf, sizeof buf, "constraint %d: unknown type %d", c, type[c]); return fail(ctx, AFSAT_E_INVALID, buf); }
        int prm = param[c];
        if (type[c] == AFSAT_OR || type[c] == AFSAT_NAE) prm = 0;
        if (type[c] == AFSAT_XOR && prm != 0 && prm != 1) { snprintf(buf, sizeof buf, "constraint %d: XOR parity must be 0 or 1", c); return fail(ctx, AFSAT_E_PARAM, buf); }
        if ((type[c] == AFSAT_ATLEAST || type[c] == AFSAT_ATMOST || type[c] == AFSAT_EXACTLY) && (prm < 0 || prm > k)) {
            snprintf(buf, sizeof buf, "constraint %d: parameter %d outside [0,%lld]", c, prm, (long long)k);
            return fail(ctx, AFSAT_E_PARAM, buf);
        }
        scratch.assign(lit_var + lo, lit_var + hi);
        for (int64_t q = lo; q < hi; ++q) {
            if (lit_var[q] < 0 || lit_var[q] >= n_vars) { snprintf(buf, sizeof buf, "constraint %d: variable %d out of range", c, lit_var[q]); return fail(ctx, AFSAT_E_VARIABLE, buf); }
            if (lit_sign[q] != 1 && lit_sign[q] != -1) { snprintf(buf, sizeof buf, "constraint %d: literal sign %d", c, lit_sign[q]); return fail(ctx, AFSAT_E_SIGN, buf); }
        }
        std::sort(scratch.begin(), scratch.end());
        if (std::adjacent_find(scratch.begin(), scratch.end()) != scratch.end()) {
            snprintf(buf, sizeof buf, "constraint %d repeats a variable", c);
            return fail(ctx, AFSAT_E_DUPLICATE, buf);
        }
        auto key = std::make_tuple((int)k, (int)type[c], prm);
        auto it = sig_id.find(key);
        if (it == sig_id.end()) it = sig_id.emplace(key, 0).first;
        (void)it;
    }
    {   // ids in (k, type, param) order so that a bucket's signatures are contiguous
        int id = 0;
        for (auto &kv : sig_id) kv.second = id++;
    }
    for (int32_t c = 0; c < n_cons; ++c) {
        const int k = (int)(row_ptr[c + 1] - row_ptr[c]);
        int prm = (type[c] == AFSAT_OR || type[c] == AFSAT_NAE) ? 0 : param[c];
        csig[c] = sig_id[std::make_tuple(k, (int)type[c], prm)];
    }

    // ---- host tables per signature -----------------------------------------------------------
    const int n_sigs = (int)sig_id.size();
    std::vector<SigDev> sigs(n_sigs);
    std::vector<double> rows;
    std::vector<float> rows2;
    std::vector<int> sig_k(n_sigs), sig_cost(n_sigs);
    for (auto &kv : sig_id) {
        AfsatSigHost hs;
        int rc = afsat_sig_build(std::get<1>(kv.first), std::get<0>(kv.first), std::get<2>(kv.first), flags, &hs);
        if (rc) return fail(ctx, rc, "signature table construction failed");
        SigDev &d = sigs[kv.second];
        memset(&d, 0, sizeof d);
        d.row_off = (int32_t)(rows.size() / 8);
        d.n_real = (int16_t)hs.n_real; d.n_cplx = (int16_t)hs.n_cplx;
        {   // discrete check scans the smaller of {satisfied, violated} counts (k_check_bits)
            const int kk = hs.k;
            auto mask_upto = [](int nbits) { return nbits >= 64 ? ~0ull : ((1ull << nbits) - 1ull); };
            const uint64_t full_lo = mask_upto(std::min(kk + 1, 64)), full_hi = kk + 1 > 64 ? mask_upto(kk + 1 - 64) : 0ull;
            const int nsat = __builtin_popcountll(hs.satmask_lo) + __builtin_popcountll(hs.satmask_hi);
            if (2 * nsat <= kk + 1) { d.scan_lo = hs.satmask_lo; d.scan_hi = hs.satmask_hi; d.scan_is_sat = 1; }
            else { d.scan_lo = ~hs.satmask_lo & full_lo; d.scan_hi = ~hs.satmask_hi & full_hi; d.scan_is_sat = 0; }
            d.k = kk;
        }
        rows.insert(rows.end(), hs.rows, hs.rows + 8 * (hs.n_real + hs.n_cplx));
        if (dtype == 32 && hs.k <= 8) {                                // staged table of the packed kernel (k <= 8)
            float r32[8 * AFSAT_MAX_POINTS], packed[AFSAT_PACK_MAX_ROWS * ROW2];
            for (int i = 0; i < 8 * (hs.n_real + hs.n_cplx); ++i) r32[i] = (float)hs.rows[i];
            int uv = 0, nu = 0, ng = 0;
            const int nrows2 = pack_rows_f2(r32, hs.n_real, hs.n_cplx, hs.k, packed, &uv, &nu, &ng);
            d.row2_off = (int32_t)(rows2.size() / ROW2);
            d.uv = (int8_t)uv; d.n_unit = (int8_t)nu; d.n_gen = (int8_t)ng;
            rows2.insert(rows2.end(), packed, packed + (size_t)nrows2 * ROW2);
        }
        sig_k[kv.second] = hs.k;
        sig_cost[kv.second] = (int)cost_of(hs.k, hs.n_real, hs.n_cplx);
    }

    // ---- bucket order: constraints sorted by (k, signature), stable ----------------------------
    std::vector<int32_t> order(n_cons);
    for (int32_t c = 0; c < n_cons; ++c) order[c] = c;
    std::stable_sort(order.begin(), order.end(), [&](int32_t a, int32_t b) { return csig[a] < csig[b]; });
    std::vector<int32_t> lits((size_t)nnz), cons_sig(n_cons);
    std::vector<int64_t> lit_off(n_cons + 1, 0);
    int64_t total_cost = 0;
    {
        int64_t w = 0;
        for (int32_t j = 0; j < n_cons; ++j) {
            const int32_t c = order[j];
            cons_sig[j] = csig[c];
            lit_off[j] = w;
            total_cost += sig_cost[csig[c]];
            for (int64_t q = row_ptr[c]; q < row_ptr[c + 1]; ++q) {
                int32_t v = lit_var[q];
                int neg = lit_sign[q] < 0;
                int32_t packed = v;
                if (fixed && fixed[v] != 0) { packed |= LIT_FIXED; neg ^= (fixed[v] < 0); }   // y = sign * (+-1)
                if (neg) packed |= LIT_NEG;
                lits[w++] = packed;
            }
        }
        lit_off[n_cons] = w;
    }

    // ---- candidate tile: X tile + G tile must stay L2-resident ------------
    const size_t esz = dtype == 32 ? 4 : 8;
    int64_t tile_w = ldb;
    {
        int64_t budget = (int64_t)104 << 20;                           // bytes of L2 for the X and G tiles (126 MB L2)
        if (const char *e = getenv("AFSAT_L2_TILE_BYTES")) { long long v = atoll(e); if (v > 0) budget = v; }
        const int64_t per_col = (int64_t)2 * n_vars * (int64_t)esz;
        // a working set within a few budgets is better left whole: the L2 misses hide behind the arithmetic, the small
        // grids of the tiles do not (cfg2 fp32, 1.58 x: 1.23 ms un-tiled vs 1.31; cfg2 fp64, 3.15 x: 2.75 vs 3.13;
        // DESIGN.md 6.5).  Beyond: equal tiles (no small remainder tile) of at most budget / per_col columns.
        if (per_col * ldb > 4 * budget) {
            const int64_t tile_max = std::max<int64_t>(64, budget / per_col / 64 * 64);
            const int64_t n_tiles = (ldb + tile_max - 1) / tile_max;
            tile_w = ((ldb + n_tiles - 1) / n_tiles + 63) / 64 * 64;
        }
        if (const char *e = getenv("AFSAT_TILE_W")) { long long v = atoll(e); if (v >= 32 && v % 32 == 0) tile_w = v; }
        tile_w = std::min<int64_t>(tile_w, ldb);
    }

    // ---- class geometry ---------------------------------------------------------------------------------
    int sm_count = 148;
    ClassGeom geom[N_CLS];
    int kmax_long = 0;
    for (int32_t j = 0; j < n_cons; ++j) { const int k = sig_k[cons_sig[j]]; if (class_of(k, dtype) == CLS_LONG) kmax_long = std::max(kmax_long, k); }
    for (int cls = 0; cls < N_CLS; ++cls) {
        ClassGeom &g = geom[cls];
        g.V = (cls == CLS_S) ? 4 : (cls == CLS_A && dtype == 32) ? AFSAT_A_V : 1;
        g.warps = CTA_WARPS;
        g.cw = 32 * g.V;
#if AFSAT_M32_PACKED
        if (cls == CLS_B && dtype == 32) {                             // packed lane-split kernel: 2 lanes x 2 candidates
            g.warps = AFSAT_M32_THREADS / 32;
            g.cw = 32;
        } else
#endif
        if (cls == CLS_LONG && dtype == 32) {                          // lane-split kernel: NS lanes per candidate
            g.warps = AFSAT_L32_THREADS / 32;
            g.cw = 32 / AFSAT_L32_NS;
#if AFSAT_L64_SPLIT
        } else if (cls == CLS_LONG) {                                  // fp64: four lanes per candidate
            g.warps = AFSAT_L64_THREADS / 32;
            g.cw = 8;
#endif
        } else if (cls == CLS_LONG) {
            const int km = long_kmax(kmax_long);
            g.warps = LONG_THREADS / 32;
            g.smem = (size_t)g.warps * (km + 2 * (km / LB)) * 32 * esz; // per warp: values [KMAX][32] + boundaries [2 KMAX/LB][32]
        }
        const int64_t cw = g.cw;
        g.Wc = std::min(g.warps, pow2_floor(std::max<int64_t>(1, (tile_w + cw - 1) / cw)));
        if ((int64_t)g.Wc * cw < tile_w && g.Wc < g.warps && (int64_t)g.Wc * cw * 2 <= tile_w + cw - 1) g.Wc *= 2;
        while (g.warps % g.Wc) --g.Wc;                                 // 12-warp CTAs: Wc x Wk must tile the CTA exactly
        g.Wk = g.warps / g.Wc;
    }

    // ---- work items: chunks of ONE signature, sized by the cost model and by the literal staging buffer ----
    std::vector<Item> items;
    int32_t cls_begin[N_CLS + 1] = {0};
    int n_buckets = 0;
    {
        int32_t j = 0;
        int cur_cls = 0, last_k = -1;
        while (j < n_cons) {
            const int sg = cons_sig[j];
            const int k = sig_k[sg];
            int32_t e = j;
            while (e < n_cons && cons_sig[e] == sg) ++e;
            if (k != last_k) { ++n_buckets; last_k = k; }
            const int cls = class_of(k, dtype);
            while (cur_cls < cls) cls_begin[++cur_cls] = (int32_t)items.size();
            const ClassGeom &g = geom[cls];
            const int64_t tiles_y = (tile_w + (int64_t)g.cw * g.Wc - 1) / ((int64_t)g.cw * g.Wc);
            const int64_t chunks_wanted = std::max<int64_t>(1, (int64_t)148 * 16 / tiles_y);
            const int64_t cost_budget = std::max<int64_t>(1, total_cost / chunks_wanted);
            const int64_t cost1 = std::max<int64_t>(1, sig_cost[sg]);
            int64_t chunk = std::max<int64_t>(g.Wk, (cost_budget + cost1 - 1) / cost1);
            chunk = std::min<int64_t>(chunk, (cls == CLS_LONG && dtype == 64 ? LONG_LIT_CHUNK : LIT_CHUNK) / k);
            chunk = std::max<int64_t>(1, chunk);
            for (int32_t s = j; s < e; s += (int32_t)chunk) {
                Item it;
                it.k = k; it.sig = sg; it.c_begin = s; it.c_end = (int32_t)std::min<int64_t>(e, s + chunk);
                it.lit_base = lit_off[s];
                it.has_fixed = 0; it.pad = 0;
                for (int64_t q = lit_off[s]; q < lit_off[it.c_end]; ++q) if (lits[q] & LIT_FIXED) { it.has_fixed = 1; break; }
                items.push_back(it);
            }
            j = e;
        }
        while (cur_cls < N_CLS) cls_begin[++cur_cls] = (int32_t)items.size();
    }

    // ---- device ----------------------------------------------------------------------------------
    ctx = new (std::nothrow) afsat_ctx;
    if (!ctx) return fail(nullptr, AFSAT_E_NOMEM, "out of host memory");
    ctx->n = n_vars; ctx->m = n_cons; ctx->B = batch; ctx->ldb = ldb; ctx->dtype = dtype; ctx->device = device;
    ctx->flags = flags; ctx->esz = dtype == 32 ? 4 : 8; ctx->nnz = nnz; ctx->n_sigs = n_sigs; ctx->n_buckets = n_buckets;
    ctx->n_items = (int32_t)items.size(); ctx->kmax_long = kmax_long; ctx->fp_instr_per_candidate = total_cost;
    ctx->tile_w = tile_w;
    memcpy(ctx->cls_begin, cls_begin, sizeof cls_begin);
    for (int cls = 0; cls < N_CLS; ++cls) ctx->geom[cls] = geom[cls];

#define CREATE_FAIL(rc_)                                   \
    do {                                                   \
        int r2_ = (rc_);                                   \
        if (r2_) { g_create_error = ctx->err; afsat_destroy(ctx); return r2_; } \
    } while (0)

    {
        int ndev = 0;
        cudaError_t e = cudaGetDeviceCount(&ndev);
        if (e != cudaSuccess || ndev <= 0 || device < 0 || device >= ndev) {
            std::string msg = std::string("no usable CUDA device ") + std::to_string(device) + " (" +
                              (e != cudaSuccess ? cudaGetErrorString(e) : "device count 0 or ordinal out of range") +
                              "); this library has no CPU fallback";
            ctx->err = msg;
            CREATE_FAIL(AFSAT_E_CUDA);
        }
    }
    CREATE_FAIL(set_device(ctx));
    {
        cudaDeviceProp prop;
        if (cudaGetDeviceProperties(&prop, device) == cudaSuccess) sm_count = prop.multiProcessorCount;
        ctx->sm_count = sm_count;
    }
    CREATE_FAIL(upload(ctx, &ctx->d_lits, lits));
    CREATE_FAIL(upload(ctx, &ctx->d_sigs, sigs));
    CREATE_FAIL(upload(ctx, &ctx->d_items, items));
    if (dtype == 32) {
        std::vector<float> r32(rows.begin(), rows.end());
        float *p = nullptr;
        CREATE_FAIL(upload(ctx, &p, r32));
        ctx->d_rows = p;
        CREATE_FAIL(upload(ctx, &ctx->d_rows2, rows2));
    } else {
        double *p = nullptr;
        CREATE_FAIL(upload(ctx, &p, rows));
        ctx->d_rows = p;
    }
    {
        std::vector<int8_t> fx(n_vars, 0);
        if (fixed) memcpy(fx.data(), fixed, n_vars);
        CREATE_FAIL(upload(ctx, &ctx->d_fixed, fx));
    }
    {
        char *g = nullptr, *fp = nullptr;
        CREATE_FAIL(dev_alloc(ctx, &g, (size_t)n_vars * tile_w * ctx->esz, true));
        ctx->d_G = g;
        CREATE_FAIL(dev_alloc(ctx, &fp, (size_t)std::max<int>(1, ctx->n_items) * ldb * ctx->esz, true));
        ctx->d_Fpart = fp;
    }
    CREATE_FAIL(dev_alloc(ctx, &ctx->d_bits, (size_t)n_vars * (size_t)(ldb / 32), true));
    CREATE_FAIL(dev_alloc(ctx, &ctx->d_satacc, (size_t)ldb, true));
    CREATE_FAIL(dev_alloc(ctx, &ctx->d_any, 2, true));
    {
        cudaError_t e = cudaStreamCreateWithFlags(&ctx->own_stream, cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ev_fork, cudaEventDisableTiming);
        for (int i = 0; i < N_CLS - 1 && e == cudaSuccess; ++i) {
            e = cudaStreamCreateWithFlags(&ctx->side_stream[i], cudaStreamNonBlocking);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ev_join[i], cudaEventDisableTiming);
        }
        if (e != cudaSuccess) { ctx->err = cudaGetErrorString(e); CREATE_FAIL(AFSAT_E_CUDA); }
    }
    *out = ctx;
    return AFSAT_OK;
}

int afsat_set_profiling(afsat_ctx *ctx, int32_t on)
{
    if (!ctx) return AFSAT_E_INVALID;
    prof_drain(ctx, false);
    ctx->prof_ns = 0.0; ctx->prof_launches = 0;
    ctx->profiling = on != 0;
    return AFSAT_OK;
}

void afsat_destroy(afsat_ctx *ctx)
{
    if (!ctx) return;
    prof_drain(ctx, false);
    cudaFree(ctx->d_lits); cudaFree(ctx->d_bits); cudaFree(ctx->d_sigs); cudaFree(ctx->d_rows); cudaFree(ctx->d_rows2);
    cudaFree(ctx->d_fixed); cudaFree(ctx->d_items); cudaFree(ctx->d_G); cudaFree(ctx->d_Fpart);
    cudaFree(ctx->d_satacc); cudaFree(ctx->d_any);
    cudaFree(ctx->ls_G); cudaFree(ctx->ls_xt); cudaFree(ctx->ls_F0); cudaFree(ctx->ls_F1); cudaFree(ctx->ls_Dpart);
    cudaFree(ctx->ls_eta); cudaFree(ctx->ls_state);
    cudaFree(ctx->dh_x); cudaFree(ctx->dh_F); cudaFree(ctx->dh_sat); cudaFree(ctx->dh_first); cudaFree(ctx->dh_sol);
    if (ctx->own_stream) cudaStreamDestroy(ctx->own_stream);
    for (int i = 0; i < N_CLS - 1; ++i) {
        if (ctx->side_stream[i]) cudaStreamDestroy(ctx->side_stream[i]);
        if (ctx->ev_join[i]) cudaEventDestroy(ctx->ev_join[i]);
    }
    if (ctx->ev_fork) cudaEventDestroy(ctx->ev_fork);
    delete ctx;
}

int afsat_eval_grad(afsat_ctx *ctx, const void *d_x, void *d_F, void *d_G, void *stream)
{
    if (!ctx) return AFSAT_E_INVALID;
    if (!d_x || (!d_F && !d_G)) return fail(ctx, AFSAT_E_INVALID, "afsat_eval_grad: NULL pointer");
    int rc = set_device(ctx);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    return ctx->dtype == 32 ? eval_grad_t<float>(ctx, (const float *)d_x, (float *)d_F, (float *)d_G, st)
                            : eval_grad_t<double>(ctx, (const double *)d_x, (double *)d_F, (double *)d_G, st);
}

int afsat_check(afsat_ctx *ctx, const void *d_x, int32_t *d_sat_count, uint8_t *d_is_solution, void *stream)
{
    if (!ctx) return AFSAT_E_INVALID;
    if (!d_x || !d_sat_count || !d_is_solution) return fail(ctx, AFSAT_E_INVALID, "afsat_check: NULL pointer");
    int rc = set_device(ctx);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    rc = ctx->dtype == 32 ? launch_pack<float>(ctx, (const float *)d_x, st) : launch_pack<double>(ctx, (const double *)d_x, st);
    if (!rc) rc = launch_check_bits(ctx, 0, ctx->ldb / 32, st);
    if (rc) return rc;
    k_check_finish<<<(ctx->B + 127) / 128, 128, 0, st>>>(ctx->d_satacc, ctx->B, ctx->m, d_sat_count, d_is_solution);
    ++ctx->launches;
    CU(cudaPeekAtLastError());
    return AFSAT_OK;
}

int afsat_step(afsat_ctx *ctx, void *d_x, double eta, int32_t n_steps, int32_t step_base, int32_t resume, void *d_F,
               int32_t *d_sat_count, uint8_t *d_is_solution, int32_t *d_first_step, int32_t *h_any_solved, void *stream)
{
    if (!ctx) return AFSAT_E_INVALID;
    if (!d_x || !d_sat_count || !d_is_solution || !d_first_step) return fail(ctx, AFSAT_E_INVALID, "afsat_step: NULL pointer");
    if (n_steps < 0) return fail(ctx, AFSAT_E_INVALID, "afsat_step: n_steps < 0");
    int rc = set_device(ctx);
    if (rc) return rc;
    int32_t *h_dev = nullptr;
    if (h_any_solved) {
        CU(cudaHostGetDevicePointer((void **)&h_dev, h_any_solved, 0));
        h_any_solved[0] = 0;
        h_any_solved[1] = -1;
    }
    cudaStream_t st = (cudaStream_t)stream;
    return ctx->dtype == 32
               ? step_t<float>(ctx, (float *)d_x, eta, n_steps, step_base, resume, (float *)d_F, d_sat_count, d_is_solution, d_first_step, h_dev, st)
               : step_t<double>(ctx, (double *)d_x, eta, n_steps, step_base, resume, (double *)d_F, d_sat_count, d_is_solution, d_first_step, h_dev, st);
}

int afsat_step_ls(afsat_ctx *ctx, void *d_x, double s_max, double beta, double c1, double delta, int32_t max_trials,
                  int32_t n_steps, int32_t step_base, int32_t resume, void *d_F, void *d_eta, int32_t *d_sat_count,
                  uint8_t *d_is_solution, int32_t *d_first_step, uint8_t *d_converged, int32_t *h_any_solved, void *stream)
{
    if (!ctx) return AFSAT_E_INVALID;
    if (!d_x || !d_sat_count || !d_is_solution || !d_first_step || !d_converged)
        return fail(ctx, AFSAT_E_INVALID, "afsat_step_ls: NULL pointer");
    if (n_steps < 0 || max_trials < 1) return fail(ctx, AFSAT_E_INVALID, "afsat_step_ls: n_steps < 0 or max_trials < 1");
    if (!(s_max > 0.0) || !(beta > 0.0 && beta < 1.0) || !(c1 >= 0.0 && c1 < 1.0) || !(delta >= 0.0))
        return fail(ctx, AFSAT_E_INVALID, "afsat_step_ls: need s_max > 0, 0 < beta < 1, 0 <= c1 < 1, delta >= 0");
    int rc = set_device(ctx);
    if (rc) return rc;
    int32_t *h_dev = nullptr;
    if (h_any_solved) {
        CU(cudaHostGetDevicePointer((void **)&h_dev, h_any_solved, 0));
        h_any_solved[0] = 0;
        h_any_solved[1] = -1;
    }
    cudaStream_t st = (cudaStream_t)stream;
    return ctx->dtype == 32
               ? step_ls_t<float>(ctx, (float *)d_x, s_max, beta, c1, delta, max_trials, n_steps, step_base, resume, (float *)d_F,
                                  d_eta, d_sat_count, d_is_solution, d_first_step, d_converged, h_dev, st)
               : step_ls_t<double>(ctx, (double *)d_x, s_max, beta, c1, delta, max_trials, n_steps, step_base, resume, (double *)d_F,
                                   d_eta, d_sat_count, d_is_solution, d_first_step, d_converged, h_dev, st);
}

int afsat_restart(afsat_ctx *ctx, void *d_x, const uint8_t *d_keep, uint64_t seed, uint32_t round, void *stream)
{
    if (!ctx) return AFSAT_E_INVALID;
    if (!d_x) return fail(ctx, AFSAT_E_INVALID, "afsat_restart: NULL pointer");
    int rc = set_device(ctx);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const unsigned gx = (unsigned)((ctx->B + CTA_THREADS - 1) / CTA_THREADS);
    const unsigned gy = (unsigned)std::min<int64_t>(ctx->n, std::max<int64_t>(1, (int64_t)ctx->sm_count * 8 / gx));
    const uint32_t lo = (uint32_t)(seed & 0xFFFFFFFFull), hi = (uint32_t)(seed >> 32);
    if (ctx->dtype == 32)
        k_restart<float><<<dim3(gx, gy), CTA_THREADS, 0, st>>>((float *)d_x, ctx->d_fixed, d_keep, lo, hi, round, ctx->n, ctx->B, ctx->ldb);
    else
        k_restart<double><<<dim3(gx, gy), CTA_THREADS, 0, st>>>((double *)d_x, ctx->d_fixed, d_keep, lo, hi, round, ctx->n, ctx->B, ctx->ldb);
    ++ctx->launches;
    CU(cudaPeekAtLastError());
    return AFSAT_OK;
}

int afsat_solve(afsat_ctx *ctx, void *d_x, double eta, int32_t steps_per_round, int32_t max_rounds, uint64_t seed,
                int32_t stop_at_first, void *d_F, int32_t *d_sat_count, uint8_t *d_is_solution, int32_t *d_first_step,
                int32_t *rounds_done, void *stream)
{
    if (!ctx) return AFSAT_E_INVALID;
    if (!d_x || !d_sat_count || !d_is_solution || !d_first_step) return fail(ctx, AFSAT_E_INVALID, "afsat_solve: NULL pointer");
    if (steps_per_round < 1 || max_rounds < 1) return fail(ctx, AFSAT_E_INVALID, "afsat_solve: steps_per_round and max_rounds must be >= 1");
    cudaStream_t st = (cudaStream_t)stream;
    int r = 0;
    for (; r < max_rounds; ++r) {
        const bool last = r + 1 == max_rounds;
        int rc = afsat_step(ctx, d_x, eta, steps_per_round, r * steps_per_round, r > 0, nullptr, d_sat_count, d_is_solution,
                            d_first_step, nullptr, stream);
        if (rc) return rc;
        int32_t any[2] = {0, -1};
        CU(cudaMemcpyAsync(any, ctx->d_any, sizeof any, cudaMemcpyDeviceToHost, st));
        CU(cudaStreamSynchronize(st));
        if ((any[0] && stop_at_first) || last) { ++r; break; }
        rc = afsat_restart(ctx, d_x, d_is_solution, seed, (uint32_t)r, stream);
        if (rc) return rc;
    }
    if (rounds_done) *rounds_done = r;
    if (d_F) return afsat_eval_grad(ctx, d_x, d_F, nullptr, stream);
    return AFSAT_OK;
}

int afsat_step_host(afsat_ctx *ctx, void *h_x, double eta, int32_t n_steps, void *h_F, int32_t *h_sat_count,
                    uint8_t *h_is_solution, int32_t *h_first_step)
{
    if (!ctx) return AFSAT_E_INVALID;
    if (!h_x) return fail(ctx, AFSAT_E_INVALID, "afsat_step_host: h_x is NULL");
    if (n_steps < 0) return fail(ctx, AFSAT_E_INVALID, "afsat_step_host: n_steps < 0");
    int rc = set_device(ctx);
    if (rc) return rc;
    const size_t xb = (size_t)ctx->n * ctx->ldb * ctx->esz;
    if (!ctx->dh_x) {
        char *px = nullptr, *pf = nullptr;
        if ((rc = dev_alloc(ctx, &px, xb))) return rc;
        ctx->dh_x = px;
        if ((rc = dev_alloc(ctx, &pf, (size_t)ctx->ldb * ctx->esz))) return rc;
        ctx->dh_F = pf;
        if ((rc = dev_alloc(ctx, &ctx->dh_sat, (size_t)ctx->ldb))) return rc;
        if ((rc = dev_alloc(ctx, &ctx->dh_first, (size_t)ctx->ldb))) return rc;
        if ((rc = dev_alloc(ctx, &ctx->dh_sol, (size_t)ctx->ldb))) return rc;
    }
    cudaStream_t st = ctx->own_stream;
    CU(cudaMemcpyAsync(ctx->dh_x, h_x, xb, cudaMemcpyHostToDevice, st));
    rc = afsat_step(ctx, ctx->dh_x, eta, n_steps, 0, 0, h_F ? ctx->dh_F : nullptr, ctx->dh_sat, ctx->dh_sol, ctx->dh_first,
                    nullptr, (void *)st);
    if (rc) return rc;
    CU(cudaMemcpyAsync(h_x, ctx->dh_x, xb, cudaMemcpyDeviceToHost, st));
    if (h_F) CU(cudaMemcpyAsync(h_F, ctx->dh_F, (size_t)ctx->B * ctx->esz, cudaMemcpyDeviceToHost, st));
    if (h_sat_count) CU(cudaMemcpyAsync(h_sat_count, ctx->dh_sat, (size_t)ctx->B * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    if (h_is_solution) CU(cudaMemcpyAsync(h_is_solution, ctx->dh_sol, (size_t)ctx->B, cudaMemcpyDeviceToHost, st));
    if (h_first_step) CU(cudaMemcpyAsync(h_first_step, ctx->dh_first, (size_t)ctx->B * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    return AFSAT_OK;
}

int64_t afsat_query(const afsat_ctx *ctx, int32_t key)
{
    if (!ctx) return -1;
    if (key == AFSAT_Q_PROFILED_EVAL_NS || key == AFSAT_Q_PROFILED_EVAL_LAUNCHES) {
        prof_drain(const_cast<afsat_ctx *>(ctx), true);
        return key == AFSAT_Q_PROFILED_EVAL_NS ? (int64_t)ctx->prof_ns : ctx->prof_launches;
    }
    switch (key) {
    case AFSAT_Q_KERNEL_LAUNCHES: return ctx->launches;
    case AFSAT_Q_NUM_SIGNATURES:  return ctx->n_sigs;
    case AFSAT_Q_NUM_BUCKETS:     return ctx->n_buckets;
    case AFSAT_Q_NNZ:             return ctx->nnz;
    case AFSAT_Q_WORKSPACE_BYTES: return (int64_t)ctx->ws_bytes;
    case AFSAT_Q_SM_COUNT:        return ctx->sm_count;
    case AFSAT_Q_FP_INSTR_PER_CANDIDATE: return ctx->fp_instr_per_candidate;
    default: return -1;
    }
}

}  // extern "C"
