// Context management, error strings, the FP64 DMMA peak probe and the host-buffer pipeline
// (include/negf.h).  No CPU fallback anywhere: negf_create fails unless a CUDA device of compute
// capability 10.x is present.
#include <stdlib.h>

#include <new>

#include "common.cuh"
#include "workspace.cuh"

extern "C" int negf_create(negf_ctx** out, int device) {
    if (!out) return NEGF_EINVAL;
    *out = nullptr;
    int count = 0;
    if (cudaGetDeviceCount(&count) != cudaSuccess || device < 0 || device >= count) return NEGF_ECUDA;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return NEGF_ECUDA;
    if (prop.major != 10) return NEGF_EUNSUPPORTED;   // kernels are built for sm_100a only
    if (cudaSetDevice(device) != cudaSuccess) return NEGF_ECUDA;
    negf_ctx* c = new (std::nothrow) negf_ctx();
    if (!c) return NEGF_EINVAL;
    c->device = device; c->stream = nullptr; c->ws = nullptr; c->ws_bytes = 0; c->last_cuda_error = 0;
    c->launches = 0; c->num_sms = prop.multiProcessorCount; c->sweep_valid = false;
    c->sw_n = c->sw_b = c->sw_ne = 0; c->sw_assembled = false; c->sw_fused = false; c->fused_small = 1;
    for (int k = 0; k < NEGF_NSIDE; k++) {
        if (cudaStreamCreateWithFlags(&c->side[k], cudaStreamNonBlocking) != cudaSuccess ||
            cudaEventCreateWithFlags(&c->ev_fork[k], cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&c->ev_join[k], cudaEventDisableTiming) != cudaSuccess) { delete c; return NEGF_ECUDA; }
    }
    if (cudaEventCreateWithFlags(&c->ev_aux, cudaEventDisableTiming) != cudaSuccess) { delete c; return NEGF_ECUDA; }
    c->graph_loops = NEGF_GRAPH_LOOPS_DEFAULT; c->gemm_3m = false; c->inv_tensor = 1; c->inv_panel = 1; c->obc_exec = nullptr; c->obc_body_launches = 0;
    for (int k = 0; k < NEGF_NGRAPH; k++) for (int q = 0; q < NEGF_GWAYS; q++) c->gslot[k][q] = {0ull, nullptr, 0, 0u};
    c->gtick = 0;
    if (cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking) != cudaSuccess) { delete c; return NEGF_ECUDA; }
    for (int k = 0; k < NEGF_MAX_ENERGY_GROUPS; k++) if (cudaEventCreateWithFlags(&c->ev_grp[k], cudaEventDisableTiming) != cudaSuccess) { delete c; return NEGF_ECUDA; }
    if (cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking) != cudaSuccess) { delete c; return NEGF_ECUDA; } c->obc_key_ws = nullptr; c->obc_key_b = c->obc_key_n = c->obc_key_ne = c->obc_key_ns = c->obc_key_maxit = 0; c->obc_key_tol = 0.0;
    c->pdl = NEGF_PDL_DEFAULT; c->in_while_body = false;
    if (const char* ev = getenv("NEGF_PDL")) { const int v = atoi(ev); if (v >= 0 && v <= 3) c->pdl = v; }   // developer override
    c->inv_lookahead = 1; c->inv_outer = 0; c->inv_side = nullptr; c->ev_inv_main = c->ev_inv_side = nullptr;
    // lowest priority: when both have CTAs pending, the caller's stream (the latency-bound panels) goes first
    int prio_lo = 0, prio_hi = 0;
    cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi);
    if (cudaStreamCreateWithPriority(&c->inv_side, cudaStreamNonBlocking, prio_lo) != cudaSuccess ||
        cudaEventCreateWithFlags(&c->ev_inv_main, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&c->ev_inv_side, cudaEventDisableTiming) != cudaSuccess) { delete c; return NEGF_ECUDA; }
    c->energy_groups = 0; c->ev_grp_fork = nullptr;
    for (int k = 0; k < NEGF_MAX_ENERGY_GROUPS; k++) { c->child[k] = nullptr; c->grp_stream[k] = nullptr; c->ev_grp_mid[k] = nullptr; }
    c->prof_on = false; c->prof_depth = 0; c->prof_last_class = -1; c->prof_last_event = nullptr;
    for (int k = 0; k < NEGF_PROF_CLASSES; k++) { c->prof_ms[k] = 0.0; c->prof_n[k] = 0; }
    if (zgemm_prepare(c) != NEGF_OK || zinv_prepare(c) != NEGF_OK || econv_prepare(c) != NEGF_OK || fused_prepare(c) != NEGF_OK) { delete c; return NEGF_ECUDA; }
    *out = c;
    return NEGF_OK;
}
extern "C" int negf_destroy(negf_ctx* ctx) {
    if (!ctx) return NEGF_EINVAL;
    for (auto& r : ctx->prof_recs) cudaEventDestroy(r.e0);
    if (ctx->prof_last_event) cudaEventDestroy(ctx->prof_last_event);
    for (int k = 0; k < NEGF_NSIDE; k++) { cudaStreamDestroy(ctx->side[k]); cudaEventDestroy(ctx->ev_fork[k]); cudaEventDestroy(ctx->ev_join[k]); }
    cudaEventDestroy(ctx->ev_aux);
    if (ctx->obc_exec) cudaGraphExecDestroy(ctx->obc_exec);
    for (int k = 0; k < NEGF_NGRAPH; k++) for (int q = 0; q < NEGF_GWAYS; q++) if (ctx->gslot[k][q].exec) cudaGraphExecDestroy(ctx->gslot[k][q].exec);
    cudaStreamDestroy(ctx->copy_stream);
    for (int k = 0; k < NEGF_MAX_ENERGY_GROUPS; k++) cudaEventDestroy(ctx->ev_grp[k]);
    cudaStreamDestroy(ctx->cap_stream);
    for (int k = 0; k < NEGF_MAX_ENERGY_GROUPS; k++) {
        if (ctx->child[k]) negf_destroy(ctx->child[k]);
        if (ctx->grp_stream[k]) cudaStreamDestroy(ctx->grp_stream[k]);
        if (ctx->ev_grp_mid[k]) cudaEventDestroy(ctx->ev_grp_mid[k]);
    }
    if (ctx->ev_grp_fork) cudaEventDestroy(ctx->ev_grp_fork);
    if (ctx->inv_side) cudaStreamDestroy(ctx->inv_side);
    if (ctx->ev_inv_main) cudaEventDestroy(ctx->ev_inv_main);
    if (ctx->ev_inv_side) cudaEventDestroy(ctx->ev_inv_side);
    delete ctx;
    return NEGF_OK;
}
extern "C" int negf_set_stream(negf_ctx* ctx, void* s) {
    if (!ctx) return NEGF_EINVAL;
    ctx->stream = (cudaStream_t)s;
    return NEGF_OK;
}
extern "C" int negf_set_workspace(negf_ctx* ctx, void* p, size_t bytes) {
    if (!ctx) return NEGF_EINVAL;
    if (p && ((uintptr_t)p & 255)) return NEGF_EINVAL;
    const bool same = p == ctx->ws && (p ? bytes : 0) == ctx->ws_bytes;
    ctx->ws = p; ctx->ws_bytes = p ? bytes : 0; ctx->sweep_valid = false;
    for (int k = 0; k < NEGF_NGRAPH; k++) for (int q = 0; q < NEGF_GWAYS; q++) ctx->gslot[k][q].key = 0;
    // the decimation WHILE graph has workspace addresses baked in: a new workspace drops it (its key also
    // holds every shape parameter the carve-up depends on, should the same address come back)
    if (!same) {
        if (ctx->obc_exec) { cudaGraphExecDestroy(ctx->obc_exec); ctx->obc_exec = nullptr; }
        ctx->obc_key_ws = nullptr;
    }
    return NEGF_OK;
}
extern "C" int negf_set_option(negf_ctx* ctx, int option, int value) {
    if (!ctx) return NEGF_EINVAL;
    if (option == NEGF_OPT_GRAPH_LOOPS) {
        if (value < 0 || value > 2) return NEGF_EINVAL;
        if (value != ctx->graph_loops && ctx->obc_exec) { cudaGraphExecDestroy(ctx->obc_exec); ctx->obc_exec = nullptr; ctx->obc_key_ws = nullptr; }
        ctx->graph_loops = value; return NEGF_OK;
    }
    if (option == NEGF_OPT_GEMM_3M) { ctx->gemm_3m = value != 0; return NEGF_OK; }
    if (option == NEGF_OPT_INV_TENSOR) { ctx->inv_tensor = value; return NEGF_OK; }
    if (option == NEGF_OPT_INV_PANEL) { ctx->inv_panel = value; return NEGF_OK; }
    if (option == NEGF_OPT_INV_LOOKAHEAD) { ctx->inv_lookahead = value; return NEGF_OK; }
    if (option == NEGF_OPT_INV_OUTER) { ctx->inv_outer = value; return NEGF_OK; }
    if (option == NEGF_OPT_PDL) {
        if (value < 0 || value > 3) return NEGF_EINVAL;
        if (value != ctx->pdl) {               // cached graphs hold the edges of the old setting
            for (int k = 0; k < NEGF_NGRAPH; k++) for (int q = 0; q < NEGF_GWAYS; q++) ctx->gslot[k][q].key = 0;
            if (ctx->obc_exec) { cudaGraphExecDestroy(ctx->obc_exec); ctx->obc_exec = nullptr; }
            ctx->obc_key_ws = nullptr;
        }
        ctx->pdl = value; return NEGF_OK;
    }
    if (option == NEGF_OPT_FUSED_SMALL) { ctx->fused_small = value; ctx->sweep_valid = false; return NEGF_OK; }
    if (option == NEGF_OPT_ENERGY_GROUPS) {
        if (value < 0 || value > NEGF_MAX_ENERGY_GROUPS) return NEGF_EINVAL;
        ctx->energy_groups = value; return NEGF_OK;
    }
    return NEGF_EINVAL;
}
extern "C" const char* negf_strerror(int code) {
    switch (code) {
        case NEGF_OK: return "ok";
        case NEGF_EINVAL: return "invalid argument";
        case NEGF_ENOWORKSPACE: return "workspace missing or too small (see negf_workspace_bytes)";
        case NEGF_EUNSUPPORTED: return "unsupported configuration or device (needs compute capability 10.x)";
        case NEGF_ECUDA: return "CUDA runtime error (see negf_last_cuda_error)";
        case NEGF_ENOSTATE: return "no retained sweep state: call negf_rgf_retarded with NEGF_KEEP_SWEEP first";
        case NEGF_ESTATICLIMIT: return "problem exceeds the static scratch of the no-allocation entry point (NEGF_STATIC_SCRATCH_BYTES)";
        default: return "unknown error code";
    }
}
extern "C" int negf_last_cuda_error(const negf_ctx* ctx) { return ctx ? ctx->last_cuda_error : 0; }
extern "C" long long negf_launch_count(const negf_ctx* ctx) { return ctx ? ctx->launches : 0; }
extern "C" long long negf_obc_graph_kernels(const negf_ctx* ctx) {
    if (!ctx) return 0;
    if (ctx->obc_exec) return ctx->obc_body_launches;
    for (int k = 0; k < NEGF_MAX_ENERGY_GROUPS; k++)
        if (ctx->child[k] && ctx->child[k]->obc_exec) return ctx->child[k]->obc_body_launches;
    return 0;
}

namespace {
// closes the open interval and folds every finished interval into the per-class totals (synchronises)
int profile_fold(negf_ctx* ctx) {
    if (ctx->prof_last_class >= 0) {
        cudaEvent_t e;
        NEGF_CUDA_CHECK(ctx, cudaEventCreate(&e));
        NEGF_CUDA_CHECK(ctx, cudaEventRecord(e, ctx->stream));
        ctx->prof_recs.push_back({ctx->prof_last_class, ctx->prof_last_event, e});
        ctx->prof_last_class = -1; ctx->prof_last_event = e;      // e is destroyed below as the chain's tail
    }
    NEGF_CUDA_CHECK(ctx, cudaStreamSynchronize(ctx->stream));
    for (auto& r : ctx->prof_recs) {
        float t = 0.f;
        NEGF_CUDA_CHECK(ctx, cudaEventElapsedTime(&t, r.e0, r.e1));
        ctx->prof_ms[r.kclass] += t;
    }
    for (auto& r : ctx->prof_recs) cudaEventDestroy(r.e0);
    ctx->prof_recs.clear();
    if (ctx->prof_last_event) { cudaEventDestroy(ctx->prof_last_event); ctx->prof_last_event = nullptr; }
    return NEGF_OK;
}
}  // namespace

extern "C" int negf_profile_enable(negf_ctx* ctx, int on) {
    if (!ctx) return NEGF_EINVAL;
    if (ctx->prof_on && !on) NEGF_TRY(profile_fold(ctx));
    ctx->prof_on = on != 0; ctx->prof_depth = 0;
    return NEGF_OK;
}
extern "C" int negf_profile_read(negf_ctx* ctx, int kclass, double* ms, long long* sites, int reset) {
    if (!ctx || kclass < 0 || kclass >= NEGF_PROF_CLASSES) return NEGF_EINVAL;
    NEGF_TRY(profile_fold(ctx));
    if (ms) *ms = ctx->prof_ms[kclass];
    if (sites) *sites = ctx->prof_n[kclass];
    if (reset) { ctx->prof_ms[kclass] = 0.0; ctx->prof_n[kclass] = 0; }
    return NEGF_OK;
}

// ---- FP64 tensor-pipe peak probe ---------------------------------------------------------------
namespace {
__global__ void __launch_bounds__(512) dmma_peak_kernel(double* out, int iters) {
    double c[8][2];
    double a = threadIdx.x * 1e-3, b = threadIdx.x * 2e-3;
#pragma unroll
    for (int i = 0; i < 8; i++) { c[i][0] = i; c[i][1] = -i; }
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int i = 0; i < 8; i++)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                         : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(a), "d"(b));
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 8; i++) s += c[i][0] + c[i][1];
    if (s == 123.456) out[0] = s;   // never true; keeps the loop alive
}
}  // namespace

extern "C" int negf_fp64_peak(negf_ctx* ctx, double ms, double* tflops) {
    if (!ctx || !tflops) return NEGF_EINVAL;
    double* d = nullptr;
    NEGF_CUDA_CHECK(ctx, cudaMalloc(&d, 64));
    cudaEvent_t e0, e1;
    NEGF_CUDA_CHECK(ctx, cudaEventCreate(&e0));
    NEGF_CUDA_CHECK(ctx, cudaEventCreate(&e1));
    const int grid = ctx->num_sms * 2, threads = 512, iters = 4000;
    const double flop_per_launch = 2.0 * 256 * 8 * (double)iters * (threads / 32) * grid;
    dmma_peak_kernel<<<grid, threads, 0, ctx->stream>>>(d, 200);
    NEGF_CUDA_CHECK(ctx, cudaStreamSynchronize(ctx->stream));
    double best = 0.0, elapsed = 0.0;
    while (elapsed < ms) {
        NEGF_CUDA_CHECK(ctx, cudaEventRecord(e0, ctx->stream));
        dmma_peak_kernel<<<grid, threads, 0, ctx->stream>>>(d, iters);
        ctx->launches++;
        NEGF_CUDA_CHECK(ctx, cudaEventRecord(e1, ctx->stream));
        NEGF_CUDA_CHECK(ctx, cudaEventSynchronize(e1));
        float t = 0.f;
        NEGF_CUDA_CHECK(ctx, cudaEventElapsedTime(&t, e0, e1));
        elapsed += t;
        double tf = flop_per_launch / (t * 1e-3) * 1e-12;
        if (tf > best) best = tf;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d);
    *tflops = best;
    return NEGF_OK;
}
