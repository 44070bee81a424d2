// afsat.cu -- C ABI (include/afsat.h) of the B200-native AFSAT hot path: context construction (validation,
// substitution of the partial assignments, bucketing by signature and length, table upload) and the launch sequences
// of afsat_eval_grad / afsat_check / afsat_step / afsat_step_ls / afsat_restart / afsat_solve / afsat_step_host.
// All arithmetic of the path runs in the kernels of afsat_kernels.cuh, afsat_split.cuh and afsat_step.cuh; the host
// tables come from precompute.cpp.  No CPU fallback exists.
#include <cuda_runtime.h>
#include <algorithm>
#include <map>
#include <mutex>
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
#include "afsat_step.cuh"

using namespace afsat;

// ---- scratch of afsat_check_static (include/afsat.h): ONE file-scope device array per GPU that loads the library.
// In HOST code the name g_static_scratch is a host-side stand-in, not a device address: never hand it to a kernel.
// afsat_static_setup resolves the device address with cudaGetSymbolAddress, once per device, and the launches get THAT.
static __device__ __align__(256) unsigned char g_static_scratch[AFSAT_STATIC_SCRATCH_BYTES];

namespace {

constexpr int STATIC_MAX_DEVICES = 64;
void *g_static_ptr[STATIC_MAX_DEVICES] = {};       // device address of g_static_scratch on device i, or null
std::mutex g_static_mutex;

thread_local std::string g_create_error;

// Length classes (one launch each per candidate tile, concurrent; one body per length, inlined into the class's kernel):
//   fp32: S  k <= 5   k_eval_f2m, FOUR candidates per lane (two packed pairs) -- the shortest constraints are issue-bound
//                     on per-constraint overhead (literal and table loads, addresses, sign masks), which a lane then
//                     pays once per four candidates
//         A  6..8     k_eval_f2m, two candidates per lane
//         B  9..20    packed lane-split kernel (two lanes x two candidates)
//         L  21..64   scalar lane-split kernel (two lanes per candidate)
//   fp64: A  k <= 8  k_eval_km (one candidate per lane);  B  9..20 / L  21..64  lane-split kernel, two / four lanes per candidate
enum { CLS_S = 0, CLS_A = 1, CLS_B = 2, CLS_LONG = 3, N_CLS = 4 };
inline int class_of(int k, int dtype)
{
    return (dtype == 32 && k <= AFSAT_S_KMAX) ? CLS_S : k <= AFSAT_A_KMAX ? CLS_A : k <= AFSAT_B_KMAX ? CLS_B : CLS_LONG;
}
constexpr int ROBUST_FROM_K = 21;       // AFSAT_FLAG_DEFAULT: robust tables from this length on (include/afsat.h)

struct ClassGeom {              // how one length class maps candidates onto a CTA
    int V = 1;                  // candidates per lane
    int cw = 32;                // candidates per warp (32 V; 32 V / NS in the lane-split kernels)
    int warps = CTA_WARPS;      // warps per CTA
    int Wc = 1, Wk = CTA_WARPS; // candidate sub-tiles x constraint groups
    int cs = 1;                 // constraints a warp walks at once (k_eval_f2m: 32 / cs lanes each)
};

// One partial assignment and the constraint table it leaves: literals of fixed variables are gone,
// constraints it decides are constants.
struct GroupPlan {
    int64_t b0 = 0, b1 = 0;     // candidates [b0, b1) (the last group also owns the padding columns up to ldb)
    int32_t *d_lits = nullptr;
    Item *d_items = nullptr;
    ConsDev *d_cons = nullptr;  // per-constraint view of the table (the one-launch step loop)
    int32_t n_items = 0, cls_begin[N_CLS + 1] = {0};
    int64_t nnz = 0;            // literals that reach a kernel
    int32_t m_live = 0;         // constraints that reach a kernel
    int32_t sat_const = 0;      // constraints the assignment satisfies outright
    double F_const = 0.0;       // decided constraints' share of F: -1 each satisfied, +1 each violated
    int64_t fp_instr = 0, flop = 0;   // cost model on the substituted table
    int32_t kmax = 0;
};

struct StepGraph {              // one captured iteration of afsat_step and what its nodes were built for
    cudaGraphExec_t exec = nullptr;
    void *x = nullptr, *sat = nullptr, *sol = nullptr, *first = nullptr, *h_any = nullptr;
    double eta = 0.0;
};

}  // namespace

struct afsat_ctx {
    int32_t n = 0, m = 0, B = 0, dtype = 32, device = 0, sm_count = 148;
    int64_t ldb = 0, nnz = 0, tile_w = 0, group_w = 0, l2_bytes = 0;
    uint32_t flags = 0;
    size_t esz = 4;
    // device tables shared by the groups
    SigDev *d_sigs = nullptr;
    void *d_rows = nullptr;
    float *d_rows2 = nullptr, *d_rows2g = nullptr; // staged tables of the packed fp32 kernel (unit rows | grouped generic rows)
    void *d_rowsg = nullptr;                       // staged tables of the grouped lane-split kernels
    int8_t *d_fixed = nullptr;                     // [n_groups][n]
    int32_t *d_sat_const = nullptr;                // [n_groups]
    std::vector<GroupPlan> groups;
    ClassGeom geom[N_CLS];
    int32_t n_sigs = 0, n_buckets = 0, max_items = 0;
    // workspace
    void *d_G = nullptr, *d_Fpart = nullptr;      // G scratch [n][tile_w]; Fpart [max_items][ldb]
    uint32_t *d_bits = nullptr;                    // sign bits [n][ldb/32]
    int32_t *d_satacc = nullptr, *d_any = nullptr; // d_any: {flag, first step, finished CTAs, step counter}
    // buffers of afsat_step_host (lazy)
    void *dh_x = nullptr, *dh_F = nullptr, *dh_Fpre = nullptr, *dh_G = nullptr;   // dh_G: full-width gradient of the pipelined un-tiled step
    int32_t *dh_sat = nullptr, *dh_first = nullptr;
    uint8_t *dh_sol = nullptr;
    cudaStream_t in_stream = nullptr, out_stream = nullptr;
    std::vector<cudaEvent_t> chunk_in, chunk_done;
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
    // how afsat_step runs its loop
    int32_t step_path = AFSAT_STEP_LAUNCHES;
    size_t small_smem = 0;
    StepGraph graph;
    bool capturing = false;
    // afsat_set_profiling: event pairs around the evaluation-kernel launches
    bool profiling = false;
    struct ProfEv { cudaEvent_t e0, e1; int cat; };
    std::vector<ProfEv> prof_events;                // cat 0: evaluation (a1-a5), 1: update (a6, a7, a9), 2: count (a8)
    double prof_ns[3] = {0.0, 0.0, 0.0};
    int64_t prof_launches[3] = {0, 0, 0};
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

inline bool misaligned(const void *p) { return ((uintptr_t)p & 15u) != 0; }

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

// model counts for one (constraint, candidate): DESIGN.md cost model
inline int64_t cost_of(int k, int n_real, int n_cplx) { return (int64_t)k * (12 * n_cplx + 4 * n_real) + 2 * n_cplx + n_real; }
inline int64_t flop_of(int k, int n_real, int n_cplx) { return (int64_t)k * (19 * n_cplx + 6 * n_real) + 4 * n_cplx + 2 * n_real; }

inline int pow2_floor(int64_t v) { int p = 1; while ((int64_t)p * 2 <= v) p *= 2; return p; }

// brackets one evaluation-kernel launch set with events when profiling is on
struct ProfScope {
    afsat_ctx *c; cudaStream_t st; int cat; cudaEvent_t e0 = nullptr, e1 = nullptr;
    ProfScope(afsat_ctx *c_, cudaStream_t st_, int cat_ = 0) : c(c_), st(st_), cat(cat_)
    {
        if (!c->profiling || c->capturing) return;
        if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) { e0 = e1 = nullptr; return; }
        cudaEventRecord(e0, st);
    }
    ~ProfScope()
    {
        if (!e0) return;
        cudaEventRecord(e1, st);
        c->prof_events.push_back({e0, e1, cat});
    }
};

void prof_drain(afsat_ctx *c, bool keep)
{
    for (auto &pr : c->prof_events) {
        if (keep && cudaEventSynchronize(pr.e1) == cudaSuccess) {
            float ms = 0.f;
            if (cudaEventElapsedTime(&ms, pr.e0, pr.e1) == cudaSuccess) { c->prof_ns[pr.cat] += (double)ms * 1e6; ++c->prof_launches[pr.cat]; }
        }
        cudaEventDestroy(pr.e0); cudaEventDestroy(pr.e1);
    }
    c->prof_events.clear();
}

// ---- kernel selection per length class ------------------------------------------------------------------------------
// grad: 0 = objective only, 1 = objective + gradient, 2 = gradient only (the packed fp32 kernel drops the contraction a3 when
// no partial objective is asked for, which is every afsat_step without F_pre; the other kernels take 2 as 1)
template <typename T>
void (*pick_kernel(int cls, int grad, bool csplit))(EvalParams<T>)
{
    using Fn = void (*)(EvalParams<T>);
    if constexpr (sizeof(T) == 4) {
        switch (cls) {
        case CLS_S:
            if (csplit) return grad == 2 ? (Fn)k_eval_f2m<1, AFSAT_S_KMAX, 2, 2, 2, true> : grad ? (Fn)k_eval_f2m<1, AFSAT_S_KMAX, 2, 1, 2, true>
                                                                                                 : (Fn)k_eval_f2m<1, AFSAT_S_KMAX, 2, 0, 2, true>;
            return grad == 2 ? (Fn)k_eval_f2m<1, AFSAT_S_KMAX, 2, 2, 2, false> : grad ? (Fn)k_eval_f2m<1, AFSAT_S_KMAX, 2, 1, 2, false>
                                                                                      : (Fn)k_eval_f2m<1, AFSAT_S_KMAX, 2, 0, 2, false>;
        case CLS_A:
            if (csplit) return grad == 2 ? (Fn)k_eval_f2m<AFSAT_S_KMAX + 1, AFSAT_A_KMAX, 1, 2, 2, true>
                                 : grad ? (Fn)k_eval_f2m<AFSAT_S_KMAX + 1, AFSAT_A_KMAX, 1, 1, 2, true>
                                        : (Fn)k_eval_f2m<AFSAT_S_KMAX + 1, AFSAT_A_KMAX, 1, 0, 2, true>;
            return grad == 2 ? (Fn)k_eval_f2m<AFSAT_S_KMAX + 1, AFSAT_A_KMAX, 1, 2, 2, false>
                      : grad ? (Fn)k_eval_f2m<AFSAT_S_KMAX + 1, AFSAT_A_KMAX, 1, 1, 2, false>
                             : (Fn)k_eval_f2m<AFSAT_S_KMAX + 1, AFSAT_A_KMAX, 1, 0, 2, false>;
        case CLS_B: return grad ? (Fn)k_eval_split<float, AFSAT_A_KMAX + 1, AFSAT_B_KMAX, 2, 2, true, AFSAT_M32_THREADS, AFSAT_M32_MINB>
                                : (Fn)k_eval_split<float, AFSAT_A_KMAX + 1, AFSAT_B_KMAX, 2, 2, false, AFSAT_M32_THREADS, AFSAT_M32_MINB>;
        default:    return grad ? (Fn)k_eval_split<float, AFSAT_L32_KMIN, AFSAT_MAX_LEN, AFSAT_L32_NS, 1, true, AFSAT_L32_THREADS, AFSAT_L32_MINB>
                                : (Fn)k_eval_split<float, AFSAT_L32_KMIN, AFSAT_MAX_LEN, AFSAT_L32_NS, 1, false, AFSAT_L32_THREADS, AFSAT_L32_MINB>;
        }
    } else {
        switch (cls) {
        case CLS_S: return nullptr;                                    // empty for fp64
        case CLS_A: return grad ? (Fn)k_eval_km<T, 1, AFSAT_A_KMAX, 1, true, 1> : (Fn)k_eval_km<T, 1, AFSAT_A_KMAX, 1, false, 1>;
        case CLS_B: return grad ? (Fn)k_eval_split<double, AFSAT_A_KMAX + 1, AFSAT_B_KMAX, 2, 1, true, AFSAT_L64_THREADS, 1>
                                : (Fn)k_eval_split<double, AFSAT_A_KMAX + 1, AFSAT_B_KMAX, 2, 1, false, AFSAT_L64_THREADS, 1>;
        default:    return grad ? (Fn)k_eval_split<double, AFSAT_L64_KMIN, AFSAT_MAX_LEN, 4, 1, true, AFSAT_L64_THREADS, 1>
                                : (Fn)k_eval_split<double, AFSAT_L64_KMIN, AFSAT_MAX_LEN, 4, 1, false, AFSAT_L64_THREADS, 1>;
        }
    }
}

// ---- launch of the evaluation kernels (a1-a5) of group gp for the candidate tile [b_begin, b_begin + width) ----
template <typename T>
int launch_eval(afsat_ctx *ctx, const GroupPlan &gp, const T *x, T *G, int64_t g_ld, int64_t g_b0, T *Fpart, int64_t b_begin,
                int64_t width, cudaStream_t st)
{
    EvalParams<T> p;
    p.x = x; p.G = G; p.g_ld = g_ld; p.g_b0 = g_b0; p.Fpart = Fpart;
    p.lits = gp.d_lits; p.sigs = ctx->d_sigs; p.rows = (const T *)ctx->d_rows; p.rows2 = ctx->d_rows2;
    p.rowsg = (const T *)ctx->d_rowsg; p.rows2g = ctx->d_rows2g;
    p.skip = ctx->cur_skip;
    p.B = ctx->B; p.ldb = ctx->ldb; p.b_begin = b_begin; p.b_end = std::min<int64_t>(b_begin + width, ctx->ldb);
    const int grad = G == nullptr ? 0 : Fpart == nullptr ? 2 : 1;
    // The length classes are independent (they only share the RED target), so their launches run
    // CONCURRENTLY: the first active class on the caller's stream, the others on forked side streams that join back.
    int n_active = 0;
    for (int cls = 0; cls < N_CLS; ++cls) n_active += gp.cls_begin[cls + 1] > gp.cls_begin[cls];
    ProfScope prof(ctx, st);                                          // brackets the whole launch set
    const bool fork = n_active > 1;
    if (fork) CU(cudaEventRecord(ctx->ev_fork, st));
    int side = 0;
    bool first_active = true;
    cudaStream_t user_st = st;
    for (int cls = 0; cls < N_CLS; ++cls) {
        const int nit = gp.cls_begin[cls + 1] - gp.cls_begin[cls];
        if (nit == 0) continue;
        st = user_st;
        int my_side = -1;
        if (fork && !first_active && side < N_CLS - 1) {
            my_side = side++;
            st = ctx->side_stream[my_side];
            CU(cudaStreamWaitEvent(st, ctx->ev_fork, 0));
        }
        first_active = false;
        const ClassGeom &g = ctx->geom[cls];
        p.items = gp.d_items + gp.cls_begin[cls];
        p.frow_base = gp.cls_begin[cls];
        p.Wc = g.Wc; p.Wk = g.Wk; p.cs = g.cs;
        const int64_t per_cta = (int64_t)g.cw * g.Wc;
        dim3 block(32 * g.warps), grid(nit, (unsigned)((width + per_cta - 1) / per_cta));
        pick_kernel<T>(cls, grad, g.cs > 1)<<<grid, block, 0, st>>>(p);
        ++ctx->launches;
        CU(cudaPeekAtLastError());
        if (my_side >= 0) {
            CU(cudaEventRecord(ctx->ev_join[my_side], st));
            CU(cudaStreamWaitEvent(user_st, ctx->ev_join[my_side], 0));
        }
    }
    return AFSAT_OK;
}

// a8 for group gp on the words [w_begin, w_end) of the sign-bit array
int launch_check_bits(afsat_ctx *ctx, const GroupPlan &gp, int64_t w_begin, int64_t w_end, int32_t *step_ctr, cudaStream_t st)
{
    if (w_end <= w_begin) return AFSAT_OK;
    CheckParams p;
    p.bits = ctx->d_bits; p.ldw = ctx->ldb / 32; p.lits = gp.d_lits; p.sigs = ctx->d_sigs; p.items = gp.d_items;
    p.satacc = ctx->d_satacc; p.B = ctx->B; p.w_begin = (int32_t)w_begin; p.w_end = (int32_t)w_end;
    p.step_ctr = step_ctr;
    const int64_t nw = w_end - w_begin;
    p.wpb = std::min(32, pow2_floor(nw));
    if (p.wpb < nw && p.wpb < 32) p.wpb *= 2;                         // cover a ragged word count in one CTA row
    p.wpb = std::min(p.wpb, 32);
    p.n_items = gp.n_items;
    const unsigned gy = (unsigned)((nw + p.wpb - 1) / p.wpb);
    dim3 grid((unsigned)std::max<int64_t>(1, std::min<int64_t>(std::max(1, gp.n_items), (int64_t)ctx->sm_count * 8 / gy)), gy);
    ProfScope prof(ctx, st, 2);
    k_check_bits<<<grid, CTA_THREADS, 0, st>>>(p);
    ++ctx->launches;
    CU(cudaPeekAtLastError());
    return AFSAT_OK;
}

// a8 over the whole batch: one launch per partial-assignment group
int check_all(afsat_ctx *ctx, bool count_step, cudaStream_t st)
{
    for (size_t g = 0; g < ctx->groups.size(); ++g) {
        const GroupPlan &gp = ctx->groups[g];
        const int64_t w1 = (g + 1 == ctx->groups.size()) ? ctx->ldb / 32 : gp.b1 / 32;
        int rc = launch_check_bits(ctx, gp, gp.b0 / 32, w1, (count_step && g == 0) ? ctx->d_any + 3 : nullptr, st);
        if (rc) return rc;
    }
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
    for (const GroupPlan &gp : ctx->groups) {
        const int64_t b1 = std::min<int64_t>(gp.b1, ctx->B);
        if (b1 <= gp.b0) continue;
        k_reduce_F<T><<<(unsigned)((b1 - gp.b0 + 31) / 32), 32 * RED_F_SLICES, 0, st>>>((const T *)ctx->d_Fpart, gp.n_items, ctx->ldb, gp.b0,
                                                                                      b1, gp.F_const, F, ctx->cur_skip);
        ++ctx->launches;
        CU(cudaPeekAtLastError());
    }
    return AFSAT_OK;
}

// the candidate tiles of a step: for every group, [b, b + w) with w <= tile_w inside the group's columns
template <typename Fn>
int for_tiles(afsat_ctx *ctx, Fn &&fn)
{
    for (size_t g = 0; g < ctx->groups.size(); ++g) {
        const GroupPlan &gp = ctx->groups[g];
        const int64_t end = (g + 1 == ctx->groups.size()) ? ctx->ldb : gp.b1;   // the last group owns the padding columns
        for (int64_t b0 = gp.b0; b0 < end && b0 < ctx->B; b0 += ctx->tile_w) {
            int rc = fn(gp, b0, std::min<int64_t>(ctx->tile_w, end - b0));
            if (rc) return rc;
        }
    }
    return AFSAT_OK;
}

template <typename T>
int eval_grad_t(afsat_ctx *ctx, const T *x, T *F, T *G, cudaStream_t st)
{
    if (G) CU(cudaMemsetAsync(G, 0, (size_t)ctx->n * ctx->ldb * sizeof(T), st));
    int rc = for_tiles(ctx, [&](const GroupPlan &gp, int64_t b0, int64_t w) {   // candidate tiles keep X/G tiles L2-resident
        return launch_eval<T>(ctx, gp, x, G, ctx->ldb, 0, F ? (T *)ctx->d_Fpart : nullptr, b0, w, st);
    });
    if (rc) return rc;
    if (G && ctx->B < ctx->ldb && (ctx->B & 3)) {                     // a lane's candidates straddle B: clear the spill
        k_zero_pad<T><<<std::min(1024, ctx->n), 128, 0, st>>>(G, ctx->n, ctx->B, ctx->ldb);
        ++ctx->launches;
        CU(cudaPeekAtLastError());
    }
    if (F) return reduce_F<T>(ctx, F, st);
    return AFSAT_OK;
}

// a6, a7, a9 on the candidate columns [b0, b0 + w) of group gp; G is the gradient array with leading dimension g_ld whose
// column 0 is candidate g_b0
template <typename T>
int launch_update(afsat_ctx *ctx, const GroupPlan &gp, T *x, T *G, int64_t g_ld, int64_t g_b0, const uint8_t *sol, double eta,
                  int64_t b0, int64_t w, cudaStream_t st)
{
    constexpr int VW = Vec16<T>::VW;
    const int tpr = std::min<int>(CTA_THREADS, pow2_floor(w / VW));   // w is a multiple of 32: tpr >= 32 / VW lanes = whole words
    const unsigned gx = (unsigned)((w / VW + tpr - 1) / tpr);
    const int rpp = CTA_THREADS / tpr;
    const unsigned gy = (unsigned)std::max<int64_t>(1, std::min<int64_t>((ctx->n + rpp * UPD_UNROLL - 1) / (rpp * UPD_UNROLL),
                                                                           (int64_t)ctx->sm_count * AFSAT_UPD_CTAS_PER_SM / gx));
    const size_t gi = &gp - ctx->groups.data();
    ProfScope prof(ctx, st, 1);
    k_update<T><<<dim3(gx, gy), CTA_THREADS, 0, st>>>(x, G, g_ld, g_b0, ctx->d_fixed + gi * (size_t)ctx->n, sol, ctx->d_bits, (T)eta,
                                                      ctx->n, ctx->B, ctx->ldb, b0, b0 + w, tpr);
    ++ctx->launches;
    CU(cudaPeekAtLastError());
    return AFSAT_OK;
}

// one iteration of Alg. 1 over the whole batch (a1-a9); step_value < 0: the step index comes from the device counter
template <typename T>
int one_iteration(afsat_ctx *ctx, T *x, double eta, int step_value, bool want_pre, int32_t *sat, uint8_t *sol, int32_t *first,
                  int32_t *h_any_dev, cudaStream_t st)
{
    const int B = ctx->B, tb = 128, gb = (B + tb - 1) / tb;
    const int64_t tw = ctx->tile_w;
    int rc = for_tiles(ctx, [&](const GroupPlan &gp, int64_t b0, int64_t w) {
        // a1-a5: gradient at X(t-1) into the (zeroed) tile scratch
        int r = launch_eval<T>(ctx, gp, x, (T *)ctx->d_G, tw, b0, want_pre ? (T *)ctx->d_Fpart : nullptr, b0, w, st);
        if (r) return r;
        // a6, a7, a9: X(t) = clamp(X(t-1) - eta G) on free variables of unsolved candidates, sign bits, G reset
        return launch_update<T>(ctx, gp, x, (T *)ctx->d_G, tw, b0, sol, eta, b0, w, st);
    });
    if (rc) return rc;
    // a8: exact count on X(t), one launch per group over its whole batch: every constraint reads the full bit rows of its
    // variables (coalesced), 1 bit per literal and candidate
    rc = check_all(ctx, step_value < 0, st);
    if (rc) return rc;
    k_flags<<<gb, tb, 0, st>>>(ctx->d_satacc, B, ctx->m, 1, step_value, step_value < 0 ? ctx->d_any + 3 : nullptr, ctx->d_sat_const,
                               ctx->group_w, (int)ctx->groups.size(), sat, sol, first, ctx->d_any, h_any_dev);
    ++ctx->launches;
    CU(cudaPeekAtLastError());
    return AFSAT_OK;
}

// the whole loop in ONE launch (k_step_small)
template <typename T>
int step_small(afsat_ctx *ctx, T *x, double eta, int n_steps, int step_base, int32_t *sat, uint8_t *sol, int32_t *first,
               int32_t *h_any_dev, cudaStream_t st)
{
    const GroupPlan &gp = ctx->groups[0];
    SmallParams<T> p;
    p.x = x; p.ldb = ctx->ldb; p.n = ctx->n; p.B = ctx->B; p.m = ctx->m; p.m_live = gp.m_live;
    p.lits = gp.d_lits; p.cons = gp.d_cons; p.sigs = ctx->d_sigs; p.rows = (const T *)ctx->d_rows; p.fixed = ctx->d_fixed;
    p.eta = (T)eta; p.n_steps = n_steps; p.step_base = step_base; p.sat_const = gp.sat_const;
    p.sat_count = sat; p.is_solution = sol; p.first_step = first; p.d_any = ctx->d_any; p.h_any = h_any_dev;
    const int threads = std::min(SMALL_THREADS, std::max(64, (gp.m_live + 31) / 32 * 32));   // thread = constraint
    k_step_small<T><<<ctx->B, threads, ctx->small_smem, st>>>(p);
    ++ctx->launches;
    CU(cudaPeekAtLastError());
    return AFSAT_OK;
}

template <typename T>
int step_t(afsat_ctx *ctx, T *x, double eta, int n_steps, int step_base, int resume, T *F, T *F_pre, int32_t *sat,
           uint8_t *sol, int32_t *first, int32_t *h_any_dev, cudaStream_t st)
{
    const int B = ctx->B, tb = 128, gb = (B + tb - 1) / tb;
    k_reset_state<<<gb, tb, 0, st>>>(B, !resume, sol, first, ctx->d_any, h_any_dev, step_base);
    ++ctx->launches;
    CU(cudaPeekAtLastError());
    int path = ctx->step_path;
    if (path == AFSAT_STEP_PERSISTENT && (F_pre || ctx->profiling)) path = AFSAT_STEP_LAUNCHES;   // F_pre is a by-product of the big kernels
    if (path == AFSAT_STEP_GRAPH && (ctx->profiling || n_steps < 3)) path = AFSAT_STEP_LAUNCHES;
    if (path == AFSAT_STEP_PERSISTENT) {
        int rc = step_small<T>(ctx, x, eta, n_steps, step_base, sat, sol, first, h_any_dev, st);
        if (rc) return rc;
    } else if (n_steps == 0) {                                        // no step: count on X as it is, mark nothing
        int rc = launch_pack<T>(ctx, x, st);
        if (!rc) rc = check_all(ctx, false, st);
        if (rc) return rc;
        k_flags<<<gb, tb, 0, st>>>(ctx->d_satacc, B, ctx->m, 0, step_base, nullptr, ctx->d_sat_const, ctx->group_w,
                                   (int)ctx->groups.size(), sat, sol, first, ctx->d_any, h_any_dev);
        ++ctx->launches;
        CU(cudaPeekAtLastError());
    } else {
        int t = 1;
        if (path == AFSAT_STEP_GRAPH) {                               // iterations 1 .. n_steps - 1 (or all): graph replays
            StepGraph &sg = ctx->graph;
            const bool stale = !sg.exec || sg.x != x || sg.sat != sat || sg.sol != sol || sg.first != first ||
                               sg.h_any != h_any_dev || sg.eta != eta;
            bool ok = true;
            if (stale) {
                if (sg.exec) { cudaGraphExecDestroy(sg.exec); sg.exec = nullptr; }
                cudaGraph_t graph = nullptr;
                const int64_t l0 = ctx->launches;
                ok = cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal) == cudaSuccess;
                if (ok) {
                    ctx->capturing = true;
                    const int rc = one_iteration<T>(ctx, x, eta, -1, false, sat, sol, first, h_any_dev, st);
                    ctx->capturing = false;
                    const cudaError_t e = cudaStreamEndCapture(st, &graph);
                    ok = rc == AFSAT_OK && e == cudaSuccess && graph &&
                         cudaGraphInstantiate(&sg.exec, graph, 0) == cudaSuccess;
                    if (graph) cudaGraphDestroy(graph);
                }
                ctx->launches = l0;                                   // captured, not launched
                if (ok) { sg.x = x; sg.sat = sat; sg.sol = sol; sg.first = first; sg.h_any = h_any_dev; sg.eta = eta; }
                else { cudaGetLastError(); sg.exec = nullptr; }
            }
            if (ok) {
                const int n_replay = F_pre ? n_steps - 1 : n_steps;
                int per_iter = 2;                                      // k_check_bits per group + k_flags
                for (const GroupPlan &gp : ctx->groups) {
                    int act = 0;
                    for (int cls = 0; cls < N_CLS; ++cls) act += gp.cls_begin[cls + 1] > gp.cls_begin[cls];
                    const int64_t end = (&gp == &ctx->groups.back()) ? ctx->ldb : gp.b1;
                    per_iter += (int)((std::min<int64_t>(end, ctx->B) - gp.b0 + ctx->tile_w - 1) / ctx->tile_w) * (act + 1);
                }
                per_iter += (int)ctx->groups.size() - 1;
                for (; t <= n_replay; ++t) {
                    CU(cudaGraphLaunch(sg.exec, st));
                    ctx->launches += per_iter;
                }
            }
        }
        for (; t <= n_steps; ++t) {
            int rc = one_iteration<T>(ctx, x, eta, path == AFSAT_STEP_GRAPH ? -1 : step_base + t, F_pre && t == n_steps, sat, sol,
                                      first, h_any_dev, st);
            if (rc) return rc;
        }
        if (F_pre) { int rc = reduce_F<T>(ctx, F_pre, st); if (rc) return rc; }
    }
    if (F) {                                                          // objective at the final X
        int rc = for_tiles(ctx, [&](const GroupPlan &gp, int64_t b0, int64_t w) {
            return launch_eval<T>(ctx, gp, x, (T *)nullptr, 0, 0, (T *)ctx->d_Fpart, b0, w, st);
        });
        if (rc) return rc;
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
    const int ng = (int)ctx->groups.size();
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
    k_reset_state<<<gb, tb, 0, st>>>(B, !resume, sol, first, ctx->d_any, h_any_dev, step_base);
    ++ctx->launches;
    if (!resume) CU(cudaMemsetAsync(conv, 0, (size_t)B, st));
    const unsigned gl = (unsigned)((ldb + CTA_THREADS - 1) / CTA_THREADS);
    const unsigned gyc = (unsigned)std::min<int64_t>(ctx->n, std::max<int64_t>(1, (int64_t)ctx->sm_count * 8 / gl));
    if (n_steps == 0) {                                               // no step: F, counts on X as it is
        k_ls_begin<<<gl, CTA_THREADS, 0, st>>>(B, ldb, sol, conv, ctx->ls_state, s_max, ctx->ls_eta);
        ++ctx->launches;
        int rc = eval_grad_t<T>(ctx, x, F0, (T *)nullptr, st);
        if (!rc) rc = launch_pack<T>(ctx, x, st);
        if (!rc) rc = check_all(ctx, false, st);
        if (rc) return rc;
        k_flags<<<gb, tb, 0, st>>>(ctx->d_satacc, B, ctx->m, 0, step_base, nullptr, ctx->d_sat_const, ctx->group_w, ng, sat, sol,
                                   first, ctx->d_any, h_any_dev);
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
            k_ls_trial<T><<<dim3(gl, LS_CHUNKS), CTA_THREADS, 0, st>>>(x, G, xt, ctx->d_fixed, ctx->group_w, ng, ctx->ls_state,
                                                                        ctx->ls_eta, ctx->ls_Dpart, ctx->n, ldb, j == 0);
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
        rc = check_all(ctx, false, st);
        if (rc) return rc;
        k_flags<<<gb, tb, 0, st>>>(ctx->d_satacc, B, ctx->m, 1, step_base + t, nullptr, ctx->d_sat_const, ctx->group_w, ng, sat,
                                   sol, first, ctx->d_any, h_any_dev);
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

// One fixed-step iteration on host buffers with the copies pipelined behind the evaluation: the batch is cut into
// candidate chunks (the tiles of a tiled step, else four), chunk c + 1 is uploaded and chunk c - 1 downloaded while
// chunk c is evaluated and updated; the count and the flags follow once for the whole batch.
template <typename T>
int step_host_pipelined(afsat_ctx *ctx, T *h_x, double eta, T *h_F_pre)
{
    cudaStream_t st = ctx->own_stream;
    const int B = ctx->B, tb = 128, gb = (B + tb - 1) / tb;
    const int64_t ldb = ctx->ldb;
    const bool tiled = ctx->tile_w < (ctx->groups.size() > 1 ? ctx->group_w : ldb);
    T *x = (T *)ctx->dh_x;
    // a chunk = a run of candidate tiles of one group, wide enough that a row of the strided host <-> device copy is a
    // few KB (512-byte rows -- one cfg4 tile -- cost the copy engines more than the pipelining gains)
    struct Chunk { const GroupPlan *gp; int64_t b0, w; };
    std::vector<Chunk> chunks;
    for (size_t g = 0; g < ctx->groups.size(); ++g) {
        const GroupPlan &gp = ctx->groups[g];
        const int64_t end = (g + 1 == ctx->groups.size()) ? ldb : gp.b1;
        int64_t cw = std::max<int64_t>(128, ((end - gp.b0 + 7) / 8 + 127) / 128 * 128);
        if (!tiled) cw = std::max<int64_t>(128, ((end - gp.b0 + 3) / 4 + 127) / 128 * 128);
        else cw = (cw + ctx->tile_w - 1) / ctx->tile_w * ctx->tile_w;                 // whole tiles
        for (int64_t b0 = gp.b0; b0 < end && b0 < B; b0 += cw) chunks.push_back({&gp, b0, std::min(cw, end - b0)});
    }
    while (ctx->chunk_in.size() < chunks.size()) {
        cudaEvent_t a, b;
        CU(cudaEventCreateWithFlags(&a, cudaEventDisableTiming));
        CU(cudaEventCreateWithFlags(&b, cudaEventDisableTiming));
        ctx->chunk_in.push_back(a); ctx->chunk_done.push_back(b);
    }
    k_reset_state<<<gb, tb, 0, st>>>(B, 1, ctx->dh_sol, ctx->dh_first, ctx->d_any, nullptr, 0);
    ++ctx->launches;
    T *G = tiled ? (T *)ctx->d_G : (T *)ctx->dh_G;                     // un-tiled: a full-width gradient
    if (!tiled) CU(cudaMemsetAsync(G, 0, (size_t)ctx->n * ldb * sizeof(T), st));
    CU(cudaEventRecord(ctx->ev_fork, st));
    CU(cudaStreamWaitEvent(ctx->in_stream, ctx->ev_fork, 0));          // uploads start after earlier work on the buffers
    CU(cudaStreamWaitEvent(ctx->out_stream, ctx->ev_fork, 0));
    for (size_t c = 0; c < chunks.size(); ++c) {
        const Chunk &ch = chunks[c];
        CU(cudaMemcpy2DAsync(x + ch.b0, ldb * sizeof(T), h_x + ch.b0, ldb * sizeof(T), ch.w * sizeof(T), ctx->n,
                             cudaMemcpyHostToDevice, ctx->in_stream));
        CU(cudaEventRecord(ctx->chunk_in[c], ctx->in_stream));
    }
    for (size_t c = 0; c < chunks.size(); ++c) {
        const Chunk &ch = chunks[c];
        CU(cudaStreamWaitEvent(st, ctx->chunk_in[c], 0));
        for (int64_t b0 = ch.b0; b0 < ch.b0 + ch.w; b0 += tiled ? ctx->tile_w : ch.w) {
            const int64_t w = tiled ? std::min<int64_t>(ctx->tile_w, ch.b0 + ch.w - b0) : ch.w;
            int rc = launch_eval<T>(ctx, *ch.gp, x, G, tiled ? ctx->tile_w : ldb, tiled ? b0 : 0, h_F_pre ? (T *)ctx->d_Fpart : nullptr,
                                    b0, w, st);
            if (!rc) rc = launch_update<T>(ctx, *ch.gp, x, G, tiled ? ctx->tile_w : ldb, tiled ? b0 : 0, ctx->dh_sol, eta, b0, w, st);
            if (rc) return rc;
        }
        CU(cudaEventRecord(ctx->chunk_done[c], st));
        CU(cudaStreamWaitEvent(ctx->out_stream, ctx->chunk_done[c], 0));
        CU(cudaMemcpy2DAsync(h_x + ch.b0, ldb * sizeof(T), x + ch.b0, ldb * sizeof(T), ch.w * sizeof(T), ctx->n,
                             cudaMemcpyDeviceToHost, ctx->out_stream));
    }
    int rc = check_all(ctx, false, st);
    if (rc) return rc;
    k_flags<<<gb, tb, 0, st>>>(ctx->d_satacc, B, ctx->m, 1, 1, nullptr, ctx->d_sat_const, ctx->group_w, (int)ctx->groups.size(),
                               ctx->dh_sat, ctx->dh_sol, ctx->dh_first, ctx->d_any, nullptr);
    ++ctx->launches;
    CU(cudaPeekAtLastError());
    if (h_F_pre) { rc = reduce_F<T>(ctx, (T *)ctx->dh_Fpre, st); if (rc) return rc; }
    return AFSAT_OK;
}

// A constraint under a partial assignment: f_T of its literals are fixed true, the k' free ones keep a
// symmetric constraint whose truth table is the original one shifted by f_T.
struct SigKey {
    int k; uint64_t lo, hi;
    bool operator<(const SigKey &o) const { return std::tie(k, lo, hi) < std::tie(o.k, o.lo, o.hi); }
};

}  // namespace

// ============================================================================================
extern "C" {

const char *afsat_version(void) { return "afsat-b200 0.2 (sm_100a)"; }

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

int afsat_host_restrict(int32_t type, int32_t k, int32_t param, int32_t f_true, int32_t f_false, int32_t *k_free, uint64_t *mask)
{
    if (!k_free || !mask) return AFSAT_E_INVALID;
    if (type < AFSAT_OR || type > AFSAT_NAE) return AFSAT_E_INVALID;
    if (k < 1 || k > AFSAT_MAX_LEN) return AFSAT_E_LENGTH;
    if (f_true < 0 || f_false < 0 || f_true + f_false > k) return AFSAT_E_INVALID;
    if (type == AFSAT_XOR && param != 0 && param != 1) return AFSAT_E_PARAM;
    if ((type == AFSAT_ATLEAST || type == AFSAT_ATMOST || type == AFSAT_EXACTLY) && (param < 0 || param > k)) return AFSAT_E_PARAM;
    const int kf = k - f_true - f_false;
    int nsat = 0;
    mask[0] = mask[1] = 0;
    for (int tau = 0; tau <= kf; ++tau)
        if (afsat_sig_satisfied(type, k, param, tau + f_true)) {
            ++nsat;
            mask[tau >> 6] |= 1ull << (tau & 63);
        }
    *k_free = kf;
    return nsat == kf + 1 ? 1 : nsat == 0 ? 2 : 0;
}

int afsat_host_tables_mask(int32_t k, uint64_t mask_lo, uint64_t mask_hi, uint32_t flags, double *table, int32_t *n_real)
{
    if (!table) return AFSAT_E_INVALID;
    AfsatSigHost s;
    int rc = afsat_sig_build_mask(k, mask_lo, mask_hi, flags & AFSAT_FLAG_ROBUST, &s);
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
    afsat_options opt;
    memset(&opt, 0, sizeof opt);
    opt.struct_size = sizeof opt;
    opt.flags = flags;
    return afsat_create_ex(out, n_vars, n_cons, row_ptr, lit_var, lit_sign, type, param, fixed, batch, ldb, dtype, device, &opt);
}

int afsat_create_ex(afsat_ctx **out, int32_t n_vars, int32_t n_cons, const int64_t *row_ptr, const int32_t *lit_var,
                    const int8_t *lit_sign, const uint8_t *type, const int32_t *param, const int8_t *fixed,
                    int32_t batch, int64_t ldb, int32_t dtype, int32_t device, const afsat_options *opt_in)
{
    afsat_ctx *ctx = nullptr;   // errors before allocation go to the thread-local message
    if (!out) return fail(ctx, AFSAT_E_INVALID, "out is NULL");
    *out = nullptr;
    afsat_options opt;
    memset(&opt, 0, sizeof opt);
    if (opt_in) {
        if (opt_in->struct_size < 8 || opt_in->struct_size > sizeof opt) return fail(ctx, AFSAT_E_INVALID, "afsat_options.struct_size");
        memcpy(&opt, opt_in, opt_in->struct_size);
    }
    const uint32_t flags = opt.flags;
    const int G = opt.n_groups <= 0 ? 1 : opt.n_groups;
    if (n_vars < 1 || n_vars > LIT_VAR) return fail(ctx, AFSAT_E_INVALID, "n_vars out of range");
    if (n_cons < 0) return fail(ctx, AFSAT_E_INVALID, "n_cons < 0");
    if (!row_ptr || (n_cons > 0 && (!type || !param))) return fail(ctx, AFSAT_E_INVALID, "NULL constraint arrays");
    if (batch < 1) return fail(ctx, AFSAT_E_INVALID, "batch must be >= 1");
    if (ldb < batch || ldb % 32 != 0) return fail(ctx, AFSAT_E_INVALID, "ldb must be >= batch and a multiple of 32");
    if (dtype != 32 && dtype != 64) return fail(ctx, AFSAT_E_INVALID, "dtype must be 32 or 64");
    if (flags & ~(uint32_t)(AFSAT_FLAG_ROBUST | AFSAT_FLAG_PAPER)) return fail(ctx, AFSAT_E_INVALID, "unknown flags");
    if ((flags & AFSAT_FLAG_ROBUST) && (flags & AFSAT_FLAG_PAPER)) return fail(ctx, AFSAT_E_INVALID, "AFSAT_FLAG_ROBUST and AFSAT_FLAG_PAPER exclude each other");
    if (G > 1 && (!fixed || batch % (32 * G) != 0))
        return fail(ctx, AFSAT_E_INVALID, "n_groups > 1 needs fixed[n_groups][n_vars] and batch % (32 n_groups) == 0");
    if (opt.tile_w < 0 || opt.tile_w % 32 != 0) return fail(ctx, AFSAT_E_INVALID, "tile_w must be a multiple of 32");
    if (opt.l2_budget_bytes < 0) return fail(ctx, AFSAT_E_INVALID, "l2_budget_bytes < 0");
    if (opt.step_path < AFSAT_STEP_AUTO || opt.step_path > AFSAT_STEP_GRAPH) return fail(ctx, AFSAT_E_INVALID, "unknown step_path");
    if (row_ptr[0] != 0) return fail(ctx, AFSAT_E_INVALID, "row_ptr[0] != 0");
    const int64_t nnz = row_ptr[n_cons];
    if (nnz > 0 && (!lit_var || !lit_sign)) return fail(ctx, AFSAT_E_INVALID, "NULL literal arrays");
    if (fixed)
        for (int64_t v = 0; v < (int64_t)G * n_vars; ++v)
            if (fixed[v] < -1 || fixed[v] > 1) return fail(ctx, AFSAT_E_SIGN, "fixed[] must be -1, 0 or +1");

    // ---- validate constraints ------------------------------------------------------------------
    std::vector<int32_t> cprm(n_cons);
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
        cprm[c] = prm;
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
    }

    // ---- device (everything above is reported even without one) ----------------------------------------
    int sm_count = 148;
    int64_t l2_bytes = (int64_t)126 << 20;
    {
        int ndev = 0;
        cudaError_t e = cudaGetDeviceCount(&ndev);
        if (e != cudaSuccess || ndev <= 0 || device < 0 || device >= ndev)
            return fail(nullptr, AFSAT_E_CUDA, std::string("no usable CUDA device ") + std::to_string(device) + " (" +
                        (e != cudaSuccess ? cudaGetErrorString(e) : "device count 0 or ordinal out of range") +
                        "); this library has no CPU fallback");
        cudaDeviceProp prop;
        e = cudaSetDevice(device);
        if (e == cudaSuccess) e = cudaGetDeviceProperties(&prop, device);
        if (e != cudaSuccess) return fail(nullptr, AFSAT_E_CUDA, std::string("cudaGetDeviceProperties: ") + cudaGetErrorString(e));
        sm_count = prop.multiProcessorCount;
        if (prop.l2CacheSize > 0) l2_bytes = prop.l2CacheSize;
    }

    // ---- substitute every partial assignment: constraint -> (k', truth table on the free literals) or a constant ----
    const int64_t group_w = G > 1 ? batch / G : ldb;
    std::map<SigKey, int> sig_id;                                // ordered by k' so that a length's signatures are contiguous
    struct Sub { SigKey key; bool live; };
    std::vector<std::vector<Sub>> subs(G, std::vector<Sub>(n_cons));
    std::vector<GroupPlan> groups(G);
    for (int g = 0; g < G; ++g) {
        const int8_t *fx = fixed ? fixed + (size_t)g * n_vars : nullptr;
        GroupPlan &gp = groups[g];
        gp.b0 = g * group_w; gp.b1 = G > 1 ? (g + 1) * group_w : batch;
        for (int32_t c = 0; c < n_cons; ++c) {
            const int k = (int)(row_ptr[c + 1] - row_ptr[c]);
            int fT = 0, kf = 0;                                        // fixed-true literals, free literals
            for (int64_t q = row_ptr[c]; q < row_ptr[c + 1]; ++q) {
                const int f = fx ? fx[lit_var[q]] : 0;
                if (!f) ++kf;
                else if ((f < 0) == (lit_sign[q] > 0)) ++fT;          // variable True and literal positive, or False and negated
            }
            uint64_t mk[2];
            int kf2 = 0;
            const int decided = afsat_host_restrict(type[c], k, cprm[c], fT, k - kf - fT, &kf2, mk);
            SigKey key{kf, mk[0], mk[1]};
            Sub &s = subs[g][c];
            s.key = key;
            s.live = decided == 0;
            if (!s.live) {                                             // decided by the partial assignment (or trivial): FE = -1 / +1
                if (decided == 1) { ++gp.sat_const; gp.F_const -= 1.0; } else gp.F_const += 1.0;
            } else {
                sig_id.emplace(key, 0);
                ++gp.m_live; gp.nnz += kf; gp.kmax = std::max(gp.kmax, kf);
            }
        }
    }
    {
        int id = 0;
        for (auto &kv : sig_id) kv.second = id++;
    }

    // ---- host tables per signature -----------------------------------------------------------
    const int n_sigs = (int)sig_id.size();
    std::vector<SigDev> sigs(n_sigs);
    std::vector<double> rows;
    std::vector<float> rows2, rows2g;
    std::vector<double> rowsg;
    std::vector<int> sig_k(n_sigs);
    std::vector<int64_t> sig_cost(n_sigs), sig_flop(n_sigs);
    for (auto &kv : sig_id) {
        AfsatSigHost hs;
        const int kk = kv.first.k;
        const bool robust = (flags & AFSAT_FLAG_ROBUST) || (!(flags & AFSAT_FLAG_PAPER) && kk >= ROBUST_FROM_K);
        int rc = afsat_sig_build_mask(kk, kv.first.lo, kv.first.hi, robust ? AFSAT_FLAG_ROBUST : 0u, &hs);
        if (rc) return fail(ctx, rc, "signature table construction failed");
        SigDev &d = sigs[kv.second];
        memset(&d, 0, sizeof d);
        d.row_off = (int32_t)(rows.size() / 8);
        d.n_real = (int16_t)hs.n_real; d.n_cplx = (int16_t)hs.n_cplx;
        {   // discrete check scans the smaller of {satisfied, violated} counts (k_check_bits)
            auto mask_upto = [](int nbits) { return nbits >= 64 ? ~0ull : ((1ull << nbits) - 1ull); };
            const uint64_t full_lo = mask_upto(std::min(kk + 1, 64)), full_hi = kk + 1 > 64 ? mask_upto(kk + 1 - 64) : 0ull;
            const int nsat = __builtin_popcountll(hs.satmask_lo) + __builtin_popcountll(hs.satmask_hi);
            if (2 * nsat <= kk + 1) { d.scan_lo = hs.satmask_lo; d.scan_hi = hs.satmask_hi; d.scan_is_sat = 1; }
            else { d.scan_lo = ~hs.satmask_lo & full_lo; d.scan_hi = ~hs.satmask_hi & full_hi; d.scan_is_sat = 0; }
            d.k = kk;
            // predicates that need no counting (k_check_bits): functions of any / all / parity of the literals
            const uint64_t slo = hs.satmask_lo, shi = hs.satmask_hi;
            auto bit_of = [&](int tau) { return (int)((tau < 64 ? slo >> tau : shi >> (tau - 64)) & 1ull); };
            bool mid_all = true, mid_none = true, odd = true, even = true;
            for (int tau = 0; tau <= kk; ++tau) {
                if (tau > 0 && tau < kk) { mid_all = mid_all && bit_of(tau); mid_none = mid_none && !bit_of(tau); }
                odd = odd && bit_of(tau) == (tau & 1); even = even && bit_of(tau) == !(tau & 1);
            }
            const int s0 = bit_of(0), sk = bit_of(kk);
            d.chk_kind = CHK_GENERAL;
            if (kk >= 2 && odd) d.chk_kind = CHK_ODD;
            else if (kk >= 2 && even) d.chk_kind = CHK_EVEN;
            else if (mid_all && !s0 && sk) d.chk_kind = CHK_OR;
            else if (mid_all && s0 && !sk) d.chk_kind = CHK_NAND;
            else if (mid_all && !s0 && !sk) d.chk_kind = CHK_NAE;
            else if (mid_none && s0 && !sk) d.chk_kind = CHK_NONE;
            else if (mid_none && !s0 && sk) d.chk_kind = CHK_ALL;
            else if (mid_none && s0 && sk && kk >= 2) d.chk_kind = CHK_EQ;
        }
        rows.insert(rows.end(), hs.rows, hs.rows + 8 * (hs.n_real + hs.n_cplx));
        if (dtype == 32 && kk <= AFSAT_A_KMAX) {                       // staged table of the packed kernel (k <= 8)
            float r32[8 * AFSAT_MAX_POINTS], packed[AFSAT_PACK_MAX_ROWS * ROW2], packedg[AFSAT_PACK_MAX_ROWS * ROW2G];
            for (int i = 0; i < 8 * (hs.n_real + hs.n_cplx); ++i) r32[i] = (float)hs.rows[i];
            int uv = 0, nu = 0, ng = 0;
            const int nrows2 = pack_rows_f2(r32, hs.rows, hs.n_real, hs.n_cplx, kk, packed, packedg, &uv, &nu, &ng);
            d.row2_off = (int32_t)(rows2.size() / ROW2);
            d.row2g_off = (int32_t)(rows2g.size() / ROW2G);
            d.uv = (int8_t)uv; d.n_unit = (int8_t)nu; d.n_gen = (int8_t)ng;
            rows2.insert(rows2.end(), packed, packed + (size_t)nrows2 * ROW2);
            rows2g.insert(rows2g.end(), packedg, packedg + (size_t)ng * ROW2G);
        }
        if (class_of(kk, dtype) == CLS_LONG || class_of(kk, dtype) == CLS_B) {   // grouped lane-split kernels
            double packed[AFSAT_MAX_POINTS * ROWG];
            const int ns = (dtype == 64 && class_of(kk, dtype) == CLS_LONG) ? 4 : 2;   // lanes per candidate (pair) of the kernel that runs kk
            d.pad = (int8_t)pack_rows_grp(hs.rows, hs.n_real + hs.n_cplx, kk, ns, packed);
            d.row2_off = (int32_t)(rowsg.size() / ROWG);
            rowsg.insert(rowsg.end(), packed, packed + (size_t)(hs.n_real + hs.n_cplx) * ROWG);
        }
        sig_k[kv.second] = kk;
        // the model counts every DFT point l < H of the constraint as it stands after substitution (R = 1 + [k odd] real)
        const int R = 1 + (kk & 1), Cc = (kk + 1) / 2 + 1 - R;
        sig_cost[kv.second] = cost_of(kk, R, Cc);
        sig_flop[kv.second] = flop_of(kk, R, Cc);
    }

    // ---- candidate tile: X tile + G tile must stay L2-resident ------------
    const size_t esz = dtype == 32 ? 4 : 8;
    const int64_t span = G > 1 ? group_w : ldb;                        // columns a tile sequence has to cover
    int64_t tile_w = span;
    {
        // X and G tiles: 13/16 of L2 (cfg4: 128 candidates, 102 MB).  Measured with ncu (profiles/r2_launches_cfg4.md): at that
        // width the tiles do NOT stay resident -- 26 GB of DRAM traffic per step where X once is 6.6 GB (the L2 is two halves,
        // one per die, and lines touched from both dies occupy both) -- while tiles of 64 candidates do; yet 128 is the
        // faster width, 17.4 against 18.0 ms per step (256: 20.0): the evaluation of such short constraints is bound by instruction
        // issue, the DRAM traffic hides under it, and the wider tile halves the per-CTA staging of the
        // literal lists.
        const int64_t budget = opt.l2_budget_bytes > 0 ? opt.l2_budget_bytes : l2_bytes / 16 * 13;
        const int64_t per_col = (int64_t)2 * n_vars * (int64_t)esz;
        // a working set within a few budgets is better left whole: the L2 misses hide behind the arithmetic, the small
        // grids of the tiles do not (cfg2 fp32, 1.58 x: 1.23 ms un-tiled vs 1.31; cfg2 fp64, 3.15 x: 2.75 vs 3.13;
        // DESIGN.md 6.5).  Beyond: equal tiles (no small remainder tile) of at most budget / per_col columns.
        if (per_col * ldb > 4 * budget) {
            const int64_t tile_max = std::max<int64_t>(64, budget / per_col / 64 * 64);
            const int64_t n_tiles = (span + tile_max - 1) / tile_max;
            tile_w = ((span + n_tiles - 1) / n_tiles + 63) / 64 * 64;
        }
        if (opt.tile_w > 0) tile_w = opt.tile_w;
        tile_w = std::max<int64_t>(32, std::min<int64_t>(tile_w, span));
    }

    // ---- class geometry ---------------------------------------------------------------------------------
    ClassGeom geom[N_CLS];
    for (int cls = 0; cls < N_CLS; ++cls) {
        ClassGeom &g = geom[cls];
        g.V = (cls == CLS_S) ? 4 : (cls == CLS_A && dtype == 32) ? 2 : 1;
        g.warps = CTA_WARPS;
        g.cw = 32 * g.V;
        if (dtype == 32 && (cls == CLS_S || cls == CLS_A))             // packed kernel: a tile narrower than a warp's candidates
            while (g.cs < 4 && g.cw / 2 >= tile_w && g.cw / 2 >= 32) { g.cs *= 2; g.cw /= 2; }   // -> several constraints per warp
        if (cls == CLS_B && dtype == 32) { g.warps = AFSAT_M32_THREADS / 32; g.cw = 32; }                 // 2 lanes x 2 candidates
        else if (cls == CLS_LONG && dtype == 32) { g.warps = AFSAT_L32_THREADS / 32; g.cw = 32 / AFSAT_L32_NS; }
        else if (cls == CLS_LONG) { g.warps = AFSAT_L64_THREADS / 32; g.cw = 8; }                         // fp64: four lanes per candidate
        else if (cls == CLS_B) { g.warps = AFSAT_L64_THREADS / 32; g.cw = 16; }                           // fp64, 9..20: two lanes per candidate
        const int64_t cw = g.cw;
        g.Wc = std::min(g.warps, pow2_floor(std::max<int64_t>(1, (tile_w + cw - 1) / cw)));
        if ((int64_t)g.Wc * cw < tile_w && g.Wc < g.warps && (int64_t)g.Wc * cw * 2 <= tile_w + cw - 1) g.Wc *= 2;
        while (g.warps % g.Wc) --g.Wc;                                 // 12-warp CTAs: Wc x Wk must tile the CTA exactly
        g.Wk = g.warps / g.Wc;
    }

    // ---- per group: bucket order, packed literals, work items ------------------------------------------------------
    std::vector<std::vector<int32_t>> g_lits(G);
    std::vector<std::vector<Item>> g_items(G);
    std::vector<std::vector<ConsDev>> g_cons(G);
    int n_buckets = 0, max_items = 1;
    for (int g = 0; g < G; ++g) {
        const int8_t *fx = fixed ? fixed + (size_t)g * n_vars : nullptr;
        GroupPlan &gp = groups[g];
        std::vector<int32_t> order;
        order.reserve(gp.m_live);
        std::vector<int32_t> csig(n_cons, -1);
        for (int32_t c = 0; c < n_cons; ++c)
            if (subs[g][c].live) { csig[c] = sig_id[subs[g][c].key]; order.push_back(c); }
        std::stable_sort(order.begin(), order.end(), [&](int32_t a, int32_t b) { return csig[a] < csig[b]; });
        std::vector<int32_t> &lits = g_lits[g];
        lits.resize((size_t)gp.nnz);
        std::vector<int64_t> lit_off(order.size() + 1, 0);
        std::vector<int32_t> cons_sig(order.size());
        int64_t w = 0;
        for (size_t j = 0; j < order.size(); ++j) {
            const int32_t c = order[j];
            cons_sig[j] = csig[c];
            lit_off[j] = w;
            gp.fp_instr += sig_cost[csig[c]]; gp.flop += sig_flop[csig[c]];
            for (int64_t q = row_ptr[c]; q < row_ptr[c + 1]; ++q) {
                const int32_t v = lit_var[q];
                if (fx && fx[v]) continue;                             // substituted
                lits[w++] = v | (lit_sign[q] < 0 ? LIT_NEG : 0);
            }
        }
        lit_off[order.size()] = w;
        if (lit_off[order.size()] < ((int64_t)1 << 31)) {
            g_cons[g].resize(order.size());
            for (size_t j = 0; j < order.size(); ++j)
                g_cons[g][j] = ConsDev{(int32_t)lit_off[j], (int16_t)cons_sig[j], (int16_t)sig_k[cons_sig[j]]};
        }
        // work items: chunks of ONE signature, sized by the cost model and by the literal staging buffer
        std::vector<Item> &items = g_items[g];
        const int32_t nc = (int32_t)order.size();
        int32_t j = 0;
        int cur_cls = 0, last_k = -1;
        while (j < nc) {
            const int sg = cons_sig[j];
            const int k = sig_k[sg];
            int32_t e = j;
            while (e < nc && cons_sig[e] == sg) ++e;
            if (g == 0 && k != last_k) { ++n_buckets; last_k = k; }
            const int cls = class_of(k, dtype);
            while (cur_cls < cls) gp.cls_begin[++cur_cls] = (int32_t)items.size();
            const ClassGeom &cg = geom[cls];
            const int64_t tiles_y = (tile_w + (int64_t)cg.cw * cg.Wc - 1) / ((int64_t)cg.cw * cg.Wc);
            const int64_t chunks_wanted = std::max<int64_t>(1, (int64_t)sm_count * 16 / tiles_y);
            const int64_t cost_budget = std::max<int64_t>(1, gp.fp_instr / chunks_wanted);
            const int64_t cost1 = std::max<int64_t>(1, sig_cost[sg]);
            int64_t chunk = std::max<int64_t>((int64_t)cg.Wk * cg.cs, (cost_budget + cost1 - 1) / cost1);
            chunk = std::min<int64_t>(chunk, LIT_CHUNK / k);
            chunk = std::max<int64_t>(1, chunk);
            for (int32_t s0 = j; s0 < e; s0 += (int32_t)chunk) {
                Item it;
                it.k = k; it.sig = sg; it.c_begin = s0; it.c_end = (int32_t)std::min<int64_t>(e, s0 + chunk);
                it.lit_base = lit_off[s0];
                it.pad0 = it.pad1 = 0;
                items.push_back(it);
            }
            j = e;
        }
        while (cur_cls < N_CLS) gp.cls_begin[++cur_cls] = (int32_t)items.size();
        gp.n_items = (int32_t)items.size();
        max_items = std::max(max_items, gp.n_items);
    }

    // ---- device ----------------------------------------------------------------------------------
    ctx = new (std::nothrow) afsat_ctx;
    if (!ctx) return fail(nullptr, AFSAT_E_NOMEM, "out of host memory");
    ctx->n = n_vars; ctx->m = n_cons; ctx->B = batch; ctx->ldb = ldb; ctx->dtype = dtype; ctx->device = device;
    ctx->flags = flags; ctx->esz = esz; ctx->nnz = nnz; ctx->n_sigs = n_sigs; ctx->n_buckets = n_buckets;
    ctx->tile_w = tile_w; ctx->group_w = group_w; ctx->sm_count = sm_count; ctx->l2_bytes = l2_bytes; ctx->max_items = max_items;
    ctx->groups = groups;
    for (int cls = 0; cls < N_CLS; ++cls) ctx->geom[cls] = geom[cls];

#define CREATE_FAIL(rc_)                                   \
    do {                                                   \
        int r2_ = (rc_);                                   \
        if (r2_) { g_create_error = ctx->err; afsat_destroy(ctx); return r2_; } \
    } while (0)

    CREATE_FAIL(set_device(ctx));
    for (int g = 0; g < G; ++g) {
        CREATE_FAIL(upload(ctx, &ctx->groups[g].d_lits, g_lits[g]));
        CREATE_FAIL(upload(ctx, &ctx->groups[g].d_items, g_items[g]));
        if (g == 0 && n_sigs < 32768) CREATE_FAIL(upload(ctx, &ctx->groups[g].d_cons, g_cons[g]));
    }
    CREATE_FAIL(upload(ctx, &ctx->d_sigs, sigs));
    if (dtype == 32) {
        std::vector<float> r32(rows.begin(), rows.end());
        float *p = nullptr;
        CREATE_FAIL(upload(ctx, &p, r32));
        ctx->d_rows = p;
        CREATE_FAIL(upload(ctx, &ctx->d_rows2, rows2));
        CREATE_FAIL(upload(ctx, &ctx->d_rows2g, rows2g));
        std::vector<float> g32(rowsg.begin(), rowsg.end());
        float *pg = nullptr;
        CREATE_FAIL(upload(ctx, &pg, g32));
        ctx->d_rowsg = pg;
    } else {
        double *p = nullptr, *pg = nullptr;
        CREATE_FAIL(upload(ctx, &p, rows));
        ctx->d_rows = p;
        CREATE_FAIL(upload(ctx, &pg, rowsg));
        ctx->d_rowsg = pg;
    }
    {
        std::vector<int8_t> fx((size_t)G * n_vars, 0);
        if (fixed) memcpy(fx.data(), fixed, fx.size());
        CREATE_FAIL(upload(ctx, &ctx->d_fixed, fx));
        std::vector<int32_t> sc(G);
        for (int g = 0; g < G; ++g) sc[g] = groups[g].sat_const;
        CREATE_FAIL(upload(ctx, &ctx->d_sat_const, sc));
    }
    {
        char *g = nullptr, *fp = nullptr;
        CREATE_FAIL(dev_alloc(ctx, &g, (size_t)n_vars * tile_w * esz, true));
        ctx->d_G = g;
        CREATE_FAIL(dev_alloc(ctx, &fp, (size_t)max_items * ldb * esz, true));
        ctx->d_Fpart = fp;
    }
    CREATE_FAIL(dev_alloc(ctx, &ctx->d_bits, (size_t)n_vars * (size_t)(ldb / 32), true));
    CREATE_FAIL(dev_alloc(ctx, &ctx->d_satacc, (size_t)ldb, true));
    CREATE_FAIL(dev_alloc(ctx, &ctx->d_any, 4, true));
    {
        cudaError_t e = cudaStreamCreateWithFlags(&ctx->own_stream, cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ev_fork, cudaEventDisableTiming);
        for (int i = 0; i < N_CLS - 1 && e == cudaSuccess; ++i) {
            e = cudaStreamCreateWithFlags(&ctx->side_stream[i], cudaStreamNonBlocking);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ev_join[i], cudaEventDisableTiming);
        }
        if (e != cudaSuccess) { ctx->err = cudaGetErrorString(e); CREATE_FAIL(AFSAT_E_CUDA); }
    }

    // ---- how afsat_step runs its loop ------------------------------------------------------------------------------------
    {
        // PERSISTENT needs: one group, every length <= 8, X and G of one candidate in shared memory
        const size_t smem = (size_t)2 * n_vars * esz;
        int dev_smem = 0;
        cudaDeviceGetAttribute(&dev_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, device);
        const bool fits = G == 1 && groups[0].kmax <= AFSAT_A_KMAX && smem + 1024 <= (size_t)dev_smem && ctx->groups[0].d_cons;
        // launch-bound when one iteration's arithmetic is shorter than its launches (~2.5 us each): model instructions
        // over the FP32 issue rate of the whole chip at ~1.9 GHz
        const double est_us = (double)groups[0].fp_instr * batch / ((double)sm_count * 128 * 1.9e3);
        int path = opt.step_path;
        if (path == AFSAT_STEP_PERSISTENT && !fits) {
            ctx->err = "AFSAT_STEP_PERSISTENT: the instance does not fit (one group, every length <= 8, X and G of a candidate in shared memory)";
            CREATE_FAIL(AFSAT_E_INVALID);
        }
        if (path == AFSAT_STEP_AUTO) {
            // (a replayed CUDA graph of one iteration, AFSAT_STEP_GRAPH, measured no faster than plain launches on cfg0 --
            // 21.0 vs 20.6 us per step: the time is kernel-to-kernel dependency latency, not host launch cost -- so it is
            // never chosen automatically)
            path = (fits && est_us < 8.0 && batch <= 8 * sm_count) ? AFSAT_STEP_PERSISTENT : AFSAT_STEP_LAUNCHES;
        }
        ctx->step_path = path;
        if (fits) {
            ctx->small_smem = smem;
            cudaError_t e = dtype == 32
                ? cudaFuncSetAttribute(k_step_small<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)
                : cudaFuncSetAttribute(k_step_small<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e != cudaSuccess) { ctx->err = std::string("cudaFuncSetAttribute(k_step_small): ") + cudaGetErrorString(e); CREATE_FAIL(AFSAT_E_CUDA); }
        }
    }
    *out = ctx;
    return AFSAT_OK;
}

int afsat_set_profiling(afsat_ctx *ctx, int32_t on)
{
    if (!ctx) return AFSAT_E_INVALID;
    prof_drain(ctx, false);
    for (int i = 0; i < 3; ++i) { ctx->prof_ns[i] = 0.0; ctx->prof_launches[i] = 0; }
    ctx->profiling = on != 0;
    return AFSAT_OK;
}

void afsat_destroy(afsat_ctx *ctx)
{
    if (!ctx) return;
    prof_drain(ctx, false);
    if (ctx->graph.exec) cudaGraphExecDestroy(ctx->graph.exec);
    for (GroupPlan &gp : ctx->groups) { cudaFree(gp.d_lits); cudaFree(gp.d_items); cudaFree(gp.d_cons); }
    cudaFree(ctx->d_bits); cudaFree(ctx->d_sigs); cudaFree(ctx->d_rows); cudaFree(ctx->d_rows2); cudaFree(ctx->d_rows2g); cudaFree(ctx->d_rowsg);
    cudaFree(ctx->d_fixed); cudaFree(ctx->d_sat_const); cudaFree(ctx->d_G); cudaFree(ctx->d_Fpart);
    cudaFree(ctx->d_satacc); cudaFree(ctx->d_any);
    cudaFree(ctx->ls_G); cudaFree(ctx->ls_xt); cudaFree(ctx->ls_F0); cudaFree(ctx->ls_F1); cudaFree(ctx->ls_Dpart);
    cudaFree(ctx->ls_eta); cudaFree(ctx->ls_state);
    cudaFree(ctx->dh_x); cudaFree(ctx->dh_F); cudaFree(ctx->dh_Fpre); cudaFree(ctx->dh_G); cudaFree(ctx->dh_sat); cudaFree(ctx->dh_first); cudaFree(ctx->dh_sol);
    for (cudaEvent_t e : ctx->chunk_in) cudaEventDestroy(e);
    for (cudaEvent_t e : ctx->chunk_done) cudaEventDestroy(e);
    if (ctx->in_stream) cudaStreamDestroy(ctx->in_stream);
    if (ctx->out_stream) cudaStreamDestroy(ctx->out_stream);
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
    if (misaligned(d_x) || misaligned(d_G)) return fail(ctx, AFSAT_E_INVALID, "afsat_eval_grad: d_x / d_G must be 16-byte aligned");
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
    if (misaligned(d_x)) return fail(ctx, AFSAT_E_INVALID, "afsat_check: d_x must be 16-byte aligned");
    int rc = set_device(ctx);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    rc = ctx->dtype == 32 ? launch_pack<float>(ctx, (const float *)d_x, st) : launch_pack<double>(ctx, (const double *)d_x, st);
    if (!rc) rc = check_all(ctx, false, st);
    if (rc) return rc;
    k_check_finish<<<(ctx->B + 127) / 128, 128, 0, st>>>(ctx->d_satacc, ctx->B, ctx->m, ctx->d_sat_const, ctx->group_w,
                                                         (int)ctx->groups.size(), d_sat_count, d_is_solution);
    ++ctx->launches;
    CU(cudaPeekAtLastError());
    return AFSAT_OK;
}

int afsat_static_setup(int32_t device)
{
    afsat_ctx *ctx = nullptr;                                         // errors go to the thread-local message
    if (device < 0 || device >= STATIC_MAX_DEVICES) return fail(ctx, AFSAT_E_INVALID, "afsat_static_setup: device ordinal out of range");
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (g_static_ptr[device]) return AFSAT_OK;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device >= ndev)
        return fail(ctx, AFSAT_E_CUDA, "afsat_static_setup: no usable CUDA device (no CPU fallback)");
    int prev = -1;
    CU(cudaGetDevice(&prev));
    CU(cudaSetDevice(device));                                        // the symbol resolves on the CURRENT device
    void *ptr = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&ptr, g_static_scratch);
    if (prev >= 0 && prev != device) cudaSetDevice(prev);
    if (e != cudaSuccess || !ptr)
        return fail(ctx, AFSAT_E_CUDA, std::string("afsat_static_setup: cudaGetSymbolAddress: ") + cudaGetErrorString(e));
    g_static_ptr[device] = ptr;
    return AFSAT_OK;
}

int afsat_check_static(afsat_ctx *ctx, const void *d_x, int32_t *d_sat_count, uint8_t *d_is_solution, void *stream)
{
    if (!ctx) return AFSAT_E_INVALID;
    if (!d_x || !d_sat_count || !d_is_solution) return fail(ctx, AFSAT_E_INVALID, "afsat_check_static: NULL pointer");
    if (misaligned(d_x)) return fail(ctx, AFSAT_E_INVALID, "afsat_check_static: d_x must be 16-byte aligned");
    // layout in the array: satacc [ldb] int32, then (256-byte aligned) the sign bits [n][ldb / 32] uint32
    const size_t ldw = (size_t)(ctx->ldb / 32);
    const size_t off_bits = ((size_t)ctx->ldb * sizeof(int32_t) + 255) / 256 * 256;
    const size_t need = off_bits + (size_t)ctx->n * ldw * sizeof(uint32_t);
    if (need > (size_t)AFSAT_STATIC_SCRATCH_BYTES) {
        char buf[200];
        snprintf(buf, sizeof buf, "afsat_check_static: this context needs %zu bytes of scratch, the static array holds %u "
                                  "(AFSAT_STATIC_SCRATCH_BYTES); use afsat_check", need, (unsigned)AFSAT_STATIC_SCRATCH_BYTES);
        return fail(ctx, AFSAT_E_NOMEM, buf);
    }
    if (ctx->device < 0 || ctx->device >= STATIC_MAX_DEVICES) return fail(ctx, AFSAT_E_INVALID, "afsat_check_static: device ordinal out of range");
    if (!g_static_ptr[ctx->device]) {                                 // not set up yet (do it BEFORE a graph capture: header)
        const int rs = afsat_static_setup(ctx->device);
        if (rs) return fail(ctx, rs, "afsat_check_static: " + g_create_error);
    }
    int rc = set_device(ctx);
    if (rc) return rc;
    unsigned char *base = (unsigned char *)g_static_ptr[ctx->device]; // the DEVICE address, never the symbol's host stand-in
    int32_t *satacc = (int32_t *)base;
    uint32_t *bits = (uint32_t *)(base + off_bits);
    cudaStream_t st = (cudaStream_t)stream;
    // the array keeps whatever the last call (of any context) left: the accumulator has to start at zero; the sign bits are
    // overwritten in full (every word of every row, padding columns as 0) before they are read
    CU(cudaMemsetAsync(satacc, 0, (size_t)ctx->ldb * sizeof(int32_t), st));
    {
        const unsigned gx = (unsigned)((ctx->ldb + CTA_THREADS - 1) / CTA_THREADS);
        const unsigned gy = (unsigned)std::min<int64_t>(ctx->n, std::max<int64_t>(1, (int64_t)ctx->sm_count * 8 / gx));
        if (ctx->dtype == 32) k_pack_signs<float><<<dim3(gx, gy), CTA_THREADS, 0, st>>>((const float *)d_x, bits, ctx->n, ctx->B, ctx->ldb);
        else k_pack_signs<double><<<dim3(gx, gy), CTA_THREADS, 0, st>>>((const double *)d_x, bits, ctx->n, ctx->B, ctx->ldb);
        ++ctx->launches;
        CU(cudaPeekAtLastError());
    }
    for (size_t g = 0; g < ctx->groups.size(); ++g) {                 // a8: one launch per partial-assignment group
        const GroupPlan &gp = ctx->groups[g];
        const int64_t w_begin = gp.b0 / 32, w_end = (g + 1 == ctx->groups.size()) ? ctx->ldb / 32 : gp.b1 / 32;
        if (w_end <= w_begin) continue;
        CheckParams p;
        p.bits = bits; p.ldw = (int64_t)ldw; p.lits = gp.d_lits; p.sigs = ctx->d_sigs; p.items = gp.d_items;
        p.satacc = satacc; p.B = ctx->B; p.w_begin = (int32_t)w_begin; p.w_end = (int32_t)w_end;
        p.step_ctr = nullptr;
        const int64_t nw = w_end - w_begin;
        p.wpb = std::min(32, pow2_floor(nw));
        if (p.wpb < nw && p.wpb < 32) p.wpb *= 2;
        p.wpb = std::min(p.wpb, 32);
        p.n_items = gp.n_items;
        const unsigned gy = (unsigned)((nw + p.wpb - 1) / p.wpb);
        dim3 grid((unsigned)std::max<int64_t>(1, std::min<int64_t>(std::max(1, gp.n_items), (int64_t)ctx->sm_count * 8 / gy)), gy);
        k_check_bits<<<grid, CTA_THREADS, 0, st>>>(p);
        ++ctx->launches;
        CU(cudaPeekAtLastError());
    }
    k_check_finish<<<(ctx->B + 127) / 128, 128, 0, st>>>(satacc, ctx->B, ctx->m, ctx->d_sat_const, ctx->group_w,
                                                         (int)ctx->groups.size(), d_sat_count, d_is_solution);
    ++ctx->launches;
    CU(cudaPeekAtLastError());
    return AFSAT_OK;
}

int afsat_step(afsat_ctx *ctx, void *d_x, double eta, int32_t n_steps, int32_t step_base, int32_t resume, void *d_F, void *d_F_pre,
               int32_t *d_sat_count, uint8_t *d_is_solution, int32_t *d_first_step, int32_t *h_any_solved, void *stream)
{
    if (!ctx) return AFSAT_E_INVALID;
    if (!d_x || !d_sat_count || !d_is_solution || !d_first_step) return fail(ctx, AFSAT_E_INVALID, "afsat_step: NULL pointer");
    if (misaligned(d_x)) return fail(ctx, AFSAT_E_INVALID, "afsat_step: d_x must be 16-byte aligned");
    if (n_steps < 0) return fail(ctx, AFSAT_E_INVALID, "afsat_step: n_steps < 0");
    int rc = set_device(ctx);
    if (rc) return rc;
    int32_t *h_dev = nullptr;
    if (h_any_solved) CU(cudaHostGetDevicePointer((void **)&h_dev, h_any_solved, 0));   // reset on the stream (k_reset_state)
    cudaStream_t st = (cudaStream_t)stream;
    return ctx->dtype == 32
               ? step_t<float>(ctx, (float *)d_x, eta, n_steps, step_base, resume, (float *)d_F, (float *)d_F_pre, d_sat_count, d_is_solution, d_first_step, h_dev, st)
               : step_t<double>(ctx, (double *)d_x, eta, n_steps, step_base, resume, (double *)d_F, (double *)d_F_pre, d_sat_count, d_is_solution, d_first_step, h_dev, st);
}

int afsat_step_ls(afsat_ctx *ctx, void *d_x, double s_max, double beta, double c1, double delta, int32_t max_trials,
                  int32_t n_steps, int32_t step_base, int32_t resume, void *d_F, void *d_eta, int32_t *d_sat_count,
                  uint8_t *d_is_solution, int32_t *d_first_step, uint8_t *d_converged, int32_t *h_any_solved, void *stream)
{
    if (!ctx) return AFSAT_E_INVALID;
    if (!d_x || !d_sat_count || !d_is_solution || !d_first_step || !d_converged)
        return fail(ctx, AFSAT_E_INVALID, "afsat_step_ls: NULL pointer");
    if (misaligned(d_x)) return fail(ctx, AFSAT_E_INVALID, "afsat_step_ls: d_x must be 16-byte aligned");
    if (n_steps < 0 || max_trials < 1) return fail(ctx, AFSAT_E_INVALID, "afsat_step_ls: n_steps < 0 or max_trials < 1");
    if (!(s_max > 0.0) || !(beta > 0.0 && beta < 1.0) || !(c1 >= 0.0 && c1 < 1.0) || !(delta >= 0.0))
        return fail(ctx, AFSAT_E_INVALID, "afsat_step_ls: need s_max > 0, 0 < beta < 1, 0 <= c1 < 1, delta >= 0");
    int rc = set_device(ctx);
    if (rc) return rc;
    int32_t *h_dev = nullptr;
    if (h_any_solved) CU(cudaHostGetDevicePointer((void **)&h_dev, h_any_solved, 0));
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
    if (misaligned(d_x)) return fail(ctx, AFSAT_E_INVALID, "afsat_restart: d_x must be 16-byte aligned");
    int rc = set_device(ctx);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const unsigned gx = (unsigned)((ctx->B + CTA_THREADS - 1) / CTA_THREADS);
    const unsigned gy = (unsigned)std::min<int64_t>(ctx->n, std::max<int64_t>(1, (int64_t)ctx->sm_count * 8 / gx));
    const uint32_t lo = (uint32_t)(seed & 0xFFFFFFFFull), hi = (uint32_t)(seed >> 32);
    const int ng = (int)ctx->groups.size();
    if (ctx->dtype == 32)
        k_restart<float><<<dim3(gx, gy), CTA_THREADS, 0, st>>>((float *)d_x, ctx->d_fixed, ctx->group_w, ng, d_keep, lo, hi, round, ctx->n, ctx->B, ctx->ldb);
    else
        k_restart<double><<<dim3(gx, gy), CTA_THREADS, 0, st>>>((double *)d_x, ctx->d_fixed, ctx->group_w, ng, d_keep, lo, hi, round, ctx->n, ctx->B, ctx->ldb);
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
        int rc = afsat_step(ctx, d_x, eta, steps_per_round, r * steps_per_round, r > 0, nullptr, nullptr, d_sat_count, d_is_solution,
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

int afsat_step_host(afsat_ctx *ctx, void *h_x, double eta, int32_t n_steps, void *h_F, void *h_F_pre, int32_t *h_sat_count,
                    uint8_t *h_is_solution, int32_t *h_first_step)
{
    if (!ctx) return AFSAT_E_INVALID;
    if (!h_x) return fail(ctx, AFSAT_E_INVALID, "afsat_step_host: h_x is NULL");
    if (n_steps < 0) return fail(ctx, AFSAT_E_INVALID, "afsat_step_host: n_steps < 0");
    int rc = set_device(ctx);
    if (rc) return rc;
    const size_t xb = (size_t)ctx->n * ctx->ldb * ctx->esz;
    if (!ctx->dh_x) {
        char *px = nullptr, *pf = nullptr, *pp = nullptr;
        if ((rc = dev_alloc(ctx, &px, xb))) return rc;
        ctx->dh_x = px;
        if ((rc = dev_alloc(ctx, &pf, (size_t)ctx->ldb * ctx->esz))) return rc;
        ctx->dh_F = pf;
        if ((rc = dev_alloc(ctx, &pp, (size_t)ctx->ldb * ctx->esz))) return rc;
        ctx->dh_Fpre = pp;
        if ((rc = dev_alloc(ctx, &ctx->dh_sat, (size_t)ctx->ldb))) return rc;
        if ((rc = dev_alloc(ctx, &ctx->dh_first, (size_t)ctx->ldb))) return rc;
        if ((rc = dev_alloc(ctx, &ctx->dh_sol, (size_t)ctx->ldb))) return rc;
        CU(cudaStreamCreateWithFlags(&ctx->in_stream, cudaStreamNonBlocking));
        CU(cudaStreamCreateWithFlags(&ctx->out_stream, cudaStreamNonBlocking));
    }
    cudaStream_t st = ctx->own_stream;
    const bool tiled = ctx->tile_w < (ctx->groups.size() > 1 ? ctx->group_w : ctx->ldb);
    // one iteration, a batch wide enough to cut: copies pipelined behind the evaluation, chunk by chunk
    const bool pipelined = n_steps == 1 && !h_F && !ctx->profiling && ctx->step_path != AFSAT_STEP_PERSISTENT &&
                           (tiled || ctx->B >= 512);
    if (pipelined && !tiled && !ctx->dh_G) {                          // un-tiled: a full-width gradient buffer
        char *pg = nullptr;
        if ((rc = dev_alloc(ctx, &pg, xb))) return rc;
        ctx->dh_G = pg;
    }
    if (pipelined) {
        rc = ctx->dtype == 32 ? step_host_pipelined<float>(ctx, (float *)h_x, eta, (float *)h_F_pre)
                              : step_host_pipelined<double>(ctx, (double *)h_x, eta, (double *)h_F_pre);
        if (rc) return rc;
    } else {
        CU(cudaMemcpyAsync(ctx->dh_x, h_x, xb, cudaMemcpyHostToDevice, st));
        rc = afsat_step(ctx, ctx->dh_x, eta, n_steps, 0, 0, h_F ? ctx->dh_F : nullptr, (h_F_pre && n_steps > 0) ? ctx->dh_Fpre : nullptr,
                        ctx->dh_sat, ctx->dh_sol, ctx->dh_first, nullptr, (void *)st);
        if (rc) return rc;
        CU(cudaMemcpyAsync(h_x, ctx->dh_x, xb, cudaMemcpyDeviceToHost, st));
    }
    if (h_F) CU(cudaMemcpyAsync(h_F, ctx->dh_F, (size_t)ctx->B * ctx->esz, cudaMemcpyDeviceToHost, st));
    if (h_F_pre && n_steps > 0) CU(cudaMemcpyAsync(h_F_pre, ctx->dh_Fpre, (size_t)ctx->B * ctx->esz, cudaMemcpyDeviceToHost, st));
    if (h_sat_count) CU(cudaMemcpyAsync(h_sat_count, ctx->dh_sat, (size_t)ctx->B * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    if (h_is_solution) CU(cudaMemcpyAsync(h_is_solution, ctx->dh_sol, (size_t)ctx->B, cudaMemcpyDeviceToHost, st));
    if (h_first_step) CU(cudaMemcpyAsync(h_first_step, ctx->dh_first, (size_t)ctx->B * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    if (pipelined) CU(cudaStreamSynchronize(ctx->out_stream));
    return AFSAT_OK;
}

int64_t afsat_query(const afsat_ctx *ctx, int32_t key)
{
    if (!ctx) return -1;
    if (key == AFSAT_Q_PROFILED_EVAL_NS || key == AFSAT_Q_PROFILED_EVAL_LAUNCHES || key == AFSAT_Q_PROFILED_UPDATE_NS ||
        key == AFSAT_Q_PROFILED_CHECK_NS) {
        prof_drain(const_cast<afsat_ctx *>(ctx), true);
        return key == AFSAT_Q_PROFILED_EVAL_NS ? (int64_t)ctx->prof_ns[0] : key == AFSAT_Q_PROFILED_UPDATE_NS ? (int64_t)ctx->prof_ns[1]
             : key == AFSAT_Q_PROFILED_CHECK_NS ? (int64_t)ctx->prof_ns[2] : ctx->prof_launches[0];
    }
    const GroupPlan &g0 = ctx->groups[0];
    switch (key) {
    case AFSAT_Q_KERNEL_LAUNCHES: return ctx->launches;
    case AFSAT_Q_NUM_SIGNATURES:  return ctx->n_sigs;
    case AFSAT_Q_NUM_BUCKETS:     return ctx->n_buckets;
    case AFSAT_Q_NNZ:             return ctx->nnz;
    case AFSAT_Q_WORKSPACE_BYTES: return (int64_t)ctx->ws_bytes;
    case AFSAT_Q_SM_COUNT:        return ctx->sm_count;
    case AFSAT_Q_FP_INSTR_PER_CANDIDATE: return g0.fp_instr;
    case AFSAT_Q_FLOP_PER_CANDIDATE: return g0.flop;
    case AFSAT_Q_NUM_GROUPS:      return (int64_t)ctx->groups.size();
    case AFSAT_Q_STEP_PATH:       return ctx->step_path;
    case AFSAT_Q_TILE_W:          return ctx->tile_w;
    case AFSAT_Q_LIVE_CONSTRAINTS: return g0.m_live;
    case AFSAT_Q_LIVE_NNZ:        return g0.nnz;
    case AFSAT_Q_DECIDED_SATISFIED: return g0.sat_const;
    case AFSAT_Q_L2_BYTES:        return ctx->l2_bytes;
    default: return -1;
    }
}

int afsat_probe_peak(int32_t device, int32_t kind, double *tflops)
{
    afsat_ctx *ctx = nullptr;
    if (!tflops || kind < 0 || kind > 5) return fail(ctx, AFSAT_E_INVALID, "afsat_probe_peak: bad arguments");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev)
        return fail(ctx, AFSAT_E_CUDA, "afsat_probe_peak: no usable CUDA device (no CPU fallback)");
    CU(cudaSetDevice(device));
    cudaDeviceProp prop;
    CU(cudaGetDeviceProperties(&prop, device));
    float *d_out = nullptr;
    CU(cudaMalloc((void **)&d_out, 64));
    cudaEvent_t e0, e1;
    CU(cudaEventCreate(&e0)); CU(cudaEventCreate(&e1));
    if (kind >= 3) {                                                  // L2 delivery rate: a 24 MB buffer, resident in either half of the L2
        const size_t bytes = (size_t)24 << 20, n_vec = bytes / sizeof(float4);
        float4 *buf = nullptr;
        CU(cudaMalloc((void **)&buf, bytes));
        CU(cudaMemset(buf, 0, bytes));
        const int iters = 400, blocks = prop.multiProcessorCount * 8;
        double best = 0.0;
        for (int rep = 0; rep < 4; ++rep) {
            CU(cudaEventRecord(e0, 0));
            if (kind == 3) k_probe_l2<0><<<blocks, 256>>>(buf, n_vec, iters, d_out);
            else if (kind == 4) k_probe_l2<1><<<blocks, 256>>>(buf, n_vec, iters, d_out);
            else k_probe_l2<2><<<blocks, 256>>>(buf, n_vec, iters, d_out);
            CU(cudaEventRecord(e1, 0));
            CU(cudaEventSynchronize(e1));
            float ms = 0.f;
            CU(cudaEventElapsedTime(&ms, e0, e1));
            if (rep > 0 && ms > 0.f) best = std::max(best, (double)bytes * iters / (ms * 1e-3) / 1e12);
        }
        cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d_out); cudaFree(buf);
        *tflops = best;                                               // TB/s
        return AFSAT_OK;
    }
    const int iters = 1 << 14, blocks = prop.multiProcessorCount * 8, threads = 256;
    double best = 0.0;
    for (int rep = 0; rep < 6; ++rep) {
        CU(cudaEventRecord(e0, 0));
        if (kind == 0) k_probe<0><<<blocks, threads>>>(d_out, iters, 1.0001f);
        else if (kind == 1) k_probe<1><<<blocks, threads>>>(d_out, iters, 1.0001f);
        else k_probe<2><<<blocks, threads>>>(d_out, iters, 1.0001f);
        CU(cudaEventRecord(e1, 0));
        CU(cudaEventSynchronize(e1));
        float ms = 0.f;
        CU(cudaEventElapsedTime(&ms, e0, e1));
        const double fma = (double)blocks * threads * iters * 8.0 * (kind == 1 ? 2.0 : 1.0);
        if (rep > 0 && ms > 0.f) best = std::max(best, 2.0 * fma / (ms * 1e-3) / 1e12);
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d_out);
    *tflops = best;
    return AFSAT_OK;
}

}  // extern "C"
