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
#include <string.h>

#include "afsat_internal.h"
#include "afsat_kernels.cuh"

using namespace afsat;

namespace {

thread_local std::string g_create_error;

enum { CLS_A = 0, CLS_B = 1, CLS_C = 2, CLS_LONG = 3, N_CLS = 4 };   // k in [1,8] [9,16] [17,24] [25,64]
inline int class_of(int k) { return k <= 8 ? CLS_A : k <= 16 ? CLS_B : k <= 24 ? CLS_C : CLS_LONG; }

}  // namespace

struct afsat_ctx {
    int32_t n = 0, m = 0, B = 0, dtype = 32, device = 0, sm_count = 148;
    int64_t ldb = 0, nnz = 0;
    uint32_t flags = 0;
    size_t esz = 4;
    // device tables
    int32_t *d_lits = nullptr, *d_cons_sig = nullptr;
    SigDev *d_sigs = nullptr;
    void *d_rows = nullptr;
    int8_t *d_fixed = nullptr;
    Item *d_items = nullptr;
    int32_t n_items = 0, cls_begin[N_CLS + 1] = {0, 0, 0, 0, 0};
    int32_t kmax_long = 0;
    int32_t n_sigs = 0, n_buckets = 0;
    int64_t fp_instr_per_candidate = 0;
    // workspace
    void *d_G = nullptr, *d_Fpart = nullptr;
    int32_t *d_satacc = nullptr, *d_any = nullptr;
    // buffers of afsat_step_host (lazy)
    void *dh_x = nullptr, *dh_F = nullptr;
    int32_t *dh_sat = nullptr, *dh_first = nullptr;
    uint8_t *dh_sol = nullptr;
    cudaStream_t own_stream = nullptr;
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

inline int warps_per_cta(const afsat_ctx *c) { return (int)std::min<int64_t>(8, c->ldb / 32); }

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

template <typename T>
int launch_eval(afsat_ctx *ctx, const T *x, T *G, T *Fpart, int32_t *satacc, bool grad, cudaStream_t st)
{
    EvalParams<T> p;
    p.x = x; p.G = G; p.Fpart = Fpart; p.satacc = satacc;
    p.lits = ctx->d_lits; p.cons_sig = ctx->d_cons_sig; p.sigs = ctx->d_sigs;
    p.rows = (const T *)ctx->d_rows; p.B = ctx->B; p.ldb = ctx->ldb;
    const int wpc = warps_per_cta(ctx);
    for (int cls = 0; cls < N_CLS; ++cls) {
        const int nit = ctx->cls_begin[cls + 1] - ctx->cls_begin[cls];
        if (nit == 0) continue;
        ProfScope prof(ctx, st);
        p.items = ctx->d_items + ctx->cls_begin[cls];
        p.item_index_base = ctx->cls_begin[cls];
        if (cls != CLS_LONG) {
            dim3 block(32 * wpc), grid(nit, (unsigned)((ctx->ldb + 32 * wpc - 1) / (32 * wpc)));
            if (cls == CLS_A) { if (grad) k_eval_reg<T, 1, 8, true><<<grid, block, 0, st>>>(p); else k_eval_reg<T, 1, 8, false><<<grid, block, 0, st>>>(p); }
            if (cls == CLS_B) { if (grad) k_eval_reg<T, 9, 16, true><<<grid, block, 0, st>>>(p); else k_eval_reg<T, 9, 16, false><<<grid, block, 0, st>>>(p); }
            if (cls == CLS_C) { if (grad) k_eval_reg<T, 17, 24, true><<<grid, block, 0, st>>>(p); else k_eval_reg<T, 17, 24, false><<<grid, block, 0, st>>>(p); }
        } else {
            const size_t per_warp = (size_t)4 * ctx->kmax_long * 32 * sizeof(T);
            int w = (int)std::max<size_t>(1, std::min<size_t>((size_t)wpc, (160 * 1024) / per_warp));
            const size_t smem = per_warp * w;
            dim3 block(32 * w), grid(nit, (unsigned)((ctx->ldb + 32 * w - 1) / (32 * w)));
            if (grad) {
                CU(cudaFuncSetAttribute(k_eval_long<T, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
                k_eval_long<T, true><<<grid, block, smem, st>>>(p, ctx->kmax_long);
            } else {
                CU(cudaFuncSetAttribute(k_eval_long<T, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
                k_eval_long<T, false><<<grid, block, smem, st>>>(p, ctx->kmax_long);
            }
        }
        ++ctx->launches;
        CU(cudaPeekAtLastError());
    }
    return AFSAT_OK;
}

template <typename T>
int launch_check(afsat_ctx *ctx, const T *x, int32_t *satacc, cudaStream_t st)
{
    if (ctx->n_items == 0) return AFSAT_OK;
    EvalParams<T> p;
    p.x = x; p.G = nullptr; p.Fpart = nullptr; p.satacc = satacc;
    p.lits = ctx->d_lits; p.cons_sig = ctx->d_cons_sig; p.sigs = ctx->d_sigs;
    p.rows = (const T *)ctx->d_rows; p.B = ctx->B; p.ldb = ctx->ldb;
    p.items = ctx->d_items; p.item_index_base = 0;
    const int wpc = warps_per_cta(ctx);
    dim3 block(32 * wpc), grid(ctx->n_items, (unsigned)((ctx->ldb + 32 * wpc - 1) / (32 * wpc)));
    k_check<T><<<grid, block, 0, st>>>(p);
    ++ctx->launches;
    CU(cudaPeekAtLastError());
    return AFSAT_OK;
}

template <typename T>
int reduce_F(afsat_ctx *ctx, T *F, cudaStream_t st)
{
    k_reduce_F<T><<<(ctx->B + 127) / 128, 128, 0, st>>>((const T *)ctx->d_Fpart, ctx->n_items, ctx->ldb, ctx->B, F);
    ++ctx->launches;
    CU(cudaPeekAtLastError());
    return AFSAT_OK;
}

template <typename T>
int eval_grad_t(afsat_ctx *ctx, const T *x, T *F, T *G, cudaStream_t st)
{
    if (G) CU(cudaMemsetAsync(G, 0, (size_t)ctx->n * ctx->ldb * sizeof(T), st));
    int rc = launch_eval<T>(ctx, x, G, F ? (T *)ctx->d_Fpart : nullptr, nullptr, G != nullptr, st);
    if (rc) return rc;
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
    CU(cudaMemsetAsync(ctx->d_satacc, 0, (size_t)ctx->ldb * sizeof(int32_t), st));
    CU(cudaMemsetAsync(ctx->d_G, 0, (size_t)ctx->n * ctx->ldb * sizeof(T), st));
    const int upd_rows = std::min(ctx->n, std::max(1, (ctx->sm_count * 16) / std::max<int>(1, (int)((ctx->ldb + 255) / 256))));
    dim3 ugrid((unsigned)((ctx->ldb + 255) / 256), upd_rows), ublock(256);
    for (int t = 1; t <= n_steps; ++t) {
        // gradient at X(t-1); from t = 2 on the same pass also counts the satisfied constraints of
        // X(t-1) (the check that Alg. 1 performs after step t-1), so the literals are read once.
        int rc = launch_eval<T>(ctx, x, (T *)ctx->d_G, nullptr, t >= 2 ? ctx->d_satacc : nullptr, true, st);
        if (rc) return rc;
        if (t >= 2) {
            k_flags<<<gb, tb, 0, st>>>(ctx->d_satacc, B, ctx->m, 0, step_base + t - 1, n_steps, sat, sol, first,
                                       ctx->d_any, h_any_dev);
            ++ctx->launches;
        }
        k_update<T><<<ugrid, ublock, 0, st>>>(x, (T *)ctx->d_G, ctx->d_fixed, sol, (T)eta, ctx->n, B, ctx->ldb);
        ++ctx->launches;
        CU(cudaPeekAtLastError());
    }
    // tail: count (and optionally F) on the final X(T)
    int rc;
    if (F) {
        rc = launch_eval<T>(ctx, x, nullptr, (T *)ctx->d_Fpart, ctx->d_satacc, false, st);
        if (!rc) rc = reduce_F<T>(ctx, F, st);
    } else {
        rc = launch_check<T>(ctx, x, ctx->d_satacc, st);
    }
    if (rc) return rc;
    k_flags<<<gb, tb, 0, st>>>(ctx->d_satacc, B, ctx->m, 1, step_base + n_steps, n_steps, sat, sol, first,
                               ctx->d_any, h_any_dev);
    ++ctx->launches;
    CU(cudaPeekAtLastError());
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
    std::vector<int> sig_k(n_sigs), sig_cost(n_sigs);
    for (auto &kv : sig_id) {
        AfsatSigHost hs;
        int rc = afsat_sig_build(std::get<1>(kv.first), std::get<0>(kv.first), std::get<2>(kv.first), flags, &hs);
        if (rc) return fail(ctx, rc, "signature table construction failed");
        SigDev &d = sigs[kv.second];
        memset(&d, 0, sizeof d);
        d.row_off = (int32_t)(rows.size() / 8);
        d.n_real = (int16_t)hs.n_real; d.n_cplx = (int16_t)hs.n_cplx;
        d.sat_lo = hs.satmask_lo; d.sat_hi = hs.satmask_hi;
        rows.insert(rows.end(), hs.rows, hs.rows + 8 * (hs.n_real + hs.n_cplx));
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

    // ---- work items: chunks of one length, sized by the cost model ------------------------------
    int sm_count = 148;
    const int wpc = (int)std::min<int64_t>(8, ldb / 32);
    const int64_t tiles_y = (ldb + 32 * wpc - 1) / (32 * wpc);
    const int64_t chunks_wanted = std::max<int64_t>(1, (int64_t)148 * 32 / tiles_y);
    const int64_t cost_budget = std::max<int64_t>(1, total_cost / chunks_wanted);
    std::vector<Item> items;
    int32_t cls_begin[N_CLS + 1] = {0, 0, 0, 0, 0};
    int n_buckets = 0, kmax_long = 0;
    {
        int32_t j = 0;
        int cur_cls = 0;
        while (j < n_cons) {
            const int k = sig_k[cons_sig[j]];
            int32_t e = j;
            int64_t bucket_cost = 0;
            while (e < n_cons && sig_k[cons_sig[e]] == k) { bucket_cost += sig_cost[cons_sig[e]]; ++e; }
            ++n_buckets;
            const int cls = class_of(k);
            while (cur_cls < cls) cls_begin[++cur_cls] = (int32_t)items.size();
            if (cls == CLS_LONG) kmax_long = std::max(kmax_long, k);
            const int64_t avg_cost = std::max<int64_t>(1, bucket_cost / (e - j));
            int64_t chunk = std::min<int64_t>(1024, std::max<int64_t>(cls == CLS_LONG ? 1 : 4, (cost_budget + avg_cost - 1) / avg_cost));
            for (int32_t s = j; s < e; s += (int32_t)chunk) {
                Item it;
                it.k = k; it.c_begin = s; it.c_end = (int32_t)std::min<int64_t>(e, s + chunk); it.pad = 0;
                it.lit_base = lit_off[s];
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
    memcpy(ctx->cls_begin, cls_begin, sizeof cls_begin);

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
    CREATE_FAIL(upload(ctx, &ctx->d_cons_sig, cons_sig));
    CREATE_FAIL(upload(ctx, &ctx->d_sigs, sigs));
    CREATE_FAIL(upload(ctx, &ctx->d_items, items));
    if (dtype == 32) {
        std::vector<float> r32(rows.begin(), rows.end());
        float *p = nullptr;
        CREATE_FAIL(upload(ctx, &p, r32));
        ctx->d_rows = p;
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
        CREATE_FAIL(dev_alloc(ctx, &g, (size_t)n_vars * ldb * ctx->esz, true));
        ctx->d_G = g;
        CREATE_FAIL(dev_alloc(ctx, &fp, (size_t)std::max<int>(1, ctx->n_items) * ldb * ctx->esz, true));
        ctx->d_Fpart = fp;
    }
    CREATE_FAIL(dev_alloc(ctx, &ctx->d_satacc, (size_t)ldb, true));
    CREATE_FAIL(dev_alloc(ctx, &ctx->d_any, 2, true));
    {
        cudaError_t e = cudaStreamCreateWithFlags(&ctx->own_stream, cudaStreamNonBlocking);
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
    cudaFree(ctx->d_lits); cudaFree(ctx->d_cons_sig); cudaFree(ctx->d_sigs); cudaFree(ctx->d_rows);
    cudaFree(ctx->d_fixed); cudaFree(ctx->d_items); cudaFree(ctx->d_G); cudaFree(ctx->d_Fpart);
    cudaFree(ctx->d_satacc); cudaFree(ctx->d_any);
    cudaFree(ctx->dh_x); cudaFree(ctx->dh_F); cudaFree(ctx->dh_sat); cudaFree(ctx->dh_first); cudaFree(ctx->dh_sol);
    if (ctx->own_stream) cudaStreamDestroy(ctx->own_stream);
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
    CU(cudaMemsetAsync(ctx->d_satacc, 0, (size_t)ctx->ldb * sizeof(int32_t), st));
    rc = ctx->dtype == 32 ? launch_check<float>(ctx, (const float *)d_x, ctx->d_satacc, st)
                          : launch_check<double>(ctx, (const double *)d_x, ctx->d_satacc, st);
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
