// Shared declarations of the CUDA side (sm_100a only).  Not included by the oracle.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include <vector>

#include "../../include/negf.h"

typedef double2 cplx;  // (x, y) = (re, im), same bytes as negf_c128
constexpr int NEGF_NSIDE = 2;
constexpr int NEGF_GWAYS = 4;     // cached argument sets per entry point (energy groups of negf_pipeline_host)
constexpr int NEGF_PDL_DEFAULT = 1;
constexpr int NEGF_GRAPH_LOOPS_DEFAULT = 2;   // negf_set_option(NEGF_OPT_GRAPH_LOOPS) at negf_create   // negf_set_option(NEGF_OPT_PDL) at negf_create
constexpr int NEGF_NGRAPH = 2;    // 0 negf_rgf_retarded, 1 negf_rgf_lesser_greater

struct negf_ctx {
    int device;
    cudaStream_t stream;          // the stream launches go to (the caller's, or temporarily a side stream)
    // side streams for independent sub-chains inside ONE call (two-sided sweeps); every call forks
    // them from the caller's stream and joins them back before it returns
    cudaStream_t side[NEGF_NSIDE];
    cudaEvent_t ev_fork[NEGF_NSIDE], ev_join[NEGF_NSIDE], ev_aux;
    void* ws;              // caller-owned workspace
    size_t ws_bytes;
    int last_cuda_error;
    long long launches;
    int num_sms;
    // retained sweep state (NEGF_KEEP_SWEEP): valid for this shape only
    bool sweep_valid;
    int sw_n, sw_b, sw_ne;
    bool sw_assembled;
    bool sw_fused;                // the retained state is the one-sided state of the resident small-block kernel
    int fused_small;              // negf_set_option(NEGF_OPT_FUSED_SMALL)
    // cached device-driven WHILE graph of the Sancho-Rubio doublings (small blocks, obc.cu)
    int graph_loops;              // negf_set_option(NEGF_OPT_GRAPH_LOOPS): 0 off, 1 = b <= 96, 2 = every block size
    bool gemm_3m;                 // negf_set_option(NEGF_OPT_GEMM_3M)
    int inv_tensor;               // negf_set_option(NEGF_OPT_INV_TENSOR)
    int inv_panel;                // negf_set_option(NEGF_OPT_INV_PANEL)
    int inv_lookahead;            // negf_set_option(NEGF_OPT_INV_LOOKAHEAD)
    int inv_outer;                // negf_set_option(NEGF_OPT_INV_OUTER); 0 = automatic
    int pdl;                      // negf_set_option(NEGF_OPT_PDL): bit 0 = chain kernels, bit 1 = also inside the WHILE graph
    cudaStream_t inv_side;        // side stream of the blocked inverse's look-ahead (zinv.cu)
    cudaEvent_t ev_inv_main, ev_inv_side;
    // cached CUDA graphs of whole calls in the latency-bound regime (same arguments twice in a row
    // -> the second call is captured, later ones replay it); one slot per entry point
    struct GraphSlot { unsigned long long key; cudaGraphExec_t exec; long long launches; unsigned used; };
    GraphSlot gslot[NEGF_NGRAPH][NEGF_GWAYS];
    unsigned gtick;
    cudaStream_t cap_stream;      // capture stream (the caller's may be the legacy default stream)
    cudaStream_t copy_stream;     // device->host copies of negf_pipeline_host
    cudaEvent_t ev_grp[NEGF_MAX_ENERGY_GROUPS];
    // concurrent energy groups of negf_pipeline_device / _host (K3): child contexts (own side streams and
    // graph caches), created on first use, each on its own stream
    int energy_groups;            // negf_set_option(NEGF_OPT_ENERGY_GROUPS); 0 = automatic
    negf_ctx* child[NEGF_MAX_ENERGY_GROUPS];
    cudaStream_t grp_stream[NEGF_MAX_ENERGY_GROUPS];
    cudaEvent_t ev_grp_fork, ev_grp_mid[NEGF_MAX_ENERGY_GROUPS];
    cudaGraphExec_t obc_exec;
    long long obc_body_launches;  // kernels in one execution of that graph's body
    // every pointer baked into that graph comes from carve_workspace(ws, n, b, ne) and the batch split ns x ne
    const void* obc_key_ws; int obc_key_b, obc_key_n, obc_key_ne, obc_key_ns, obc_key_maxit; double obc_key_tol;
    // optional per-kernel-class timing (negf_profile_enable): event pairs around every launch site
    bool prof_on;
    int prof_depth;
    struct ProfRec { int kclass; cudaEvent_t e0, e1; };
    std::vector<ProfRec> prof_recs;     // e1 of a record is e0 of the next one
    int prof_last_class; cudaEvent_t prof_last_event;
    double prof_ms[NEGF_PROF_CLASSES];
    long long prof_n[NEGF_PROF_CLASSES];
    bool in_while_body;           // the decimation WHILE graph's body is being captured
    bool pdl_now() const { return !prof_on && (in_while_body ? (pdl & 2) != 0 : (pdl & 1) != 0); }
};

// Per-class device time when profiling is on: ONE event is recorded on the stream whenever the kernel
// class of the next launch site differs from the previous one, so consecutive launches of a class form
// one interval (two event records per launch would cost more than the small kernels they bracket).
// Nested scopes (the GEMMs inside the blocked inverse) are charged to the outermost class.  While
// profiling, the side streams are not used (StreamFork), so the intervals never overlap.
struct ProfScope {
    negf_ctx* c;
    ProfScope(negf_ctx* ctx, int kclass) : c(ctx) {
        if (!c->prof_on) return;
        if (c->prof_depth++ == 0 && kclass != c->prof_last_class) {
            cudaEvent_t e;
            cudaEventCreate(&e);
            cudaEventRecord(e, c->stream);
            if (c->prof_last_class >= 0) c->prof_recs.push_back({c->prof_last_class, c->prof_last_event, e});
            c->prof_last_class = kclass; c->prof_last_event = e;
        }
    }
    ~ProfScope() { if (c->prof_on) c->prof_depth--; }
};

#define NEGF_CUDA_CHECK(ctx, expr)                                  \
    do {                                                            \
        cudaError_t _e = (expr);                                    \
        if (_e != cudaSuccess) {                                    \
            (ctx)->last_cuda_error = (int)_e;                       \
            return NEGF_ECUDA;                                      \
        }                                                           \
    } while (0)

#define NEGF_COUNT_LAUNCH(ctx)                                      \
    do {                                                            \
        (ctx)->launches++;                                          \
        if ((ctx)->prof_on && (ctx)->prof_last_class >= 0) (ctx)->prof_n[(ctx)->prof_last_class]++; \
    } while (0)

#define NEGF_LAUNCH_CHECK(ctx)                                      \
    do {                                                            \
        NEGF_COUNT_LAUNCH(ctx);                                     \
        cudaError_t _e = cudaGetLastError();                        \
        if (_e != cudaSuccess) {                                    \
            (ctx)->last_cuda_error = (int)_e;                       \
            return NEGF_ECUDA;                                      \
        }                                                           \
    } while (0)

// Programmatic dependent launch (sm_90+): a kernel of the latency-bound chains (K2 small tiles, the one-CTA
// inverses, the decimation step) is launched with the programmatic-stream-serialization attribute, so its
// CTAs are placed on the SMs while the previous kernel of the stream drains; it calls pdl_wait() before its
// first global-memory access (returns when the previous kernel has completed and its writes are visible) and
// pdl_trigger() right after (so at most one waiting kernel is resident behind the running one).  Both are
// no-ops in a kernel launched without the attribute.  Only kernels that call pdl_wait() may be launched this way.
#ifdef __CUDACC__
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
#endif
template <class... KArgs, class... Args>
inline cudaError_t launch_chain(negf_ctx* ctx, void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, Args&&... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = ctx->stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = (ctx->pdl_now() ? 1 : 0);
    return cudaLaunchKernelEx(&cfg, kern, static_cast<KArgs>(args)...);
}

#define NEGF_TRY(expr)                   \
    do {                                 \
        int _r = (expr);                 \
        if (_r != NEGF_OK) return _r;    \
    } while (0)

__host__ __device__ inline cplx cmake(double r, double i) { cplx c; c.x = r; c.y = i; return c; }
__device__ __forceinline__ cplx cadd(cplx a, cplx b) { return cmake(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ cplx csub(cplx a, cplx b) { return cmake(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ cplx cmul(cplx a, cplx b) {
    return cmake(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
__device__ __forceinline__ cplx cconj(cplx a) { return cmake(a.x, -a.y); }
__device__ __forceinline__ cplx cneg(cplx a) { return cmake(-a.x, -a.y); }
// c += a*b
__device__ __forceinline__ void cfma(cplx& c, cplx a, cplx b) {
    c.x = fma(a.x, b.x, c.x); c.x = fma(-a.y, b.y, c.x);
    c.y = fma(a.x, b.y, c.y); c.y = fma(a.y, b.x, c.y);
}
// c -= a*b
__device__ __forceinline__ void cfms(cplx& c, cplx a, cplx b) {
    c.x = fma(-a.x, b.x, c.x); c.x = fma(a.y, b.y, c.x);
    c.y = fma(-a.x, b.y, c.y); c.y = fma(-a.y, b.x, c.y);
}
// robust 1/a (Smith) -- pivots are O(1) here but keep it safe
__device__ __forceinline__ cplx crecip(cplx a) {
    if (fabs(a.x) >= fabs(a.y)) {
        double r = a.y / a.x, d = a.x + a.y * r;
        return cmake(1.0 / d, -r / d);
    } else {
        double r = a.x / a.y, d = a.x * r + a.y;
        return cmake(r / d, -1.0 / d);
    }
}
__device__ __forceinline__ double cabs1(cplx a) { return fabs(a.x) + fabs(a.y); }

static inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// Fork / join of the side streams and redirection of ctx->stream (restored by the destructor on
// every exit path).  main = the caller's stream as it was when the guard was built.
struct StreamFork {
    negf_ctx* c; cudaStream_t main;
    explicit StreamFork(negf_ctx* ctx) : c(ctx), main(ctx->stream) {}
    ~StreamFork() { c->stream = main; }
    void use_main() { c->stream = main; }
    void use_side(int k) { if (!c->prof_on) c->stream = c->side[k]; }
    // side k starts after everything enqueued on `from` so far (default: main)
    cudaError_t fork(int k) {
        if (c->prof_on) return cudaSuccess;
        cudaError_t e = cudaEventRecord(c->ev_fork[k], main);
        return e != cudaSuccess ? e : cudaStreamWaitEvent(c->side[k], c->ev_fork[k], 0);
    }
    // main continues after everything enqueued on side k so far
    cudaError_t join(int k) {
        if (c->prof_on) return cudaSuccess;
        cudaError_t e = cudaEventRecord(c->ev_join[k], c->side[k]);
        return e != cudaSuccess ? e : cudaStreamWaitEvent(main, c->ev_join[k], 0);
    }
    // side k waits for everything enqueued on main so far (mid-call dependency)
    cudaError_t side_waits_main(int k) {
        if (c->prof_on) return cudaSuccess;
        cudaError_t e = cudaEventRecord(c->ev_aux, main);
        return e != cudaSuccess ? e : cudaStreamWaitEvent(c->side[k], c->ev_aux, 0);
    }
};

// FNV-1a over argument bytes: the key of a cached call graph
struct KeyHash {
    unsigned long long h = 1469598103934665603ull;
    void add(const void* p, size_t n) {
        const unsigned char* c = (const unsigned char*)p;
        for (size_t i = 0; i < n; i++) { h ^= c[i]; h *= 1099511628211ull; }
    }
    template <class T> void val(const T& v) { add(&v, sizeof(T)); }
};

// Runs `body` (which only enqueues work on ctx->stream) directly, or - when the same key was seen on the
// previous call - captures it once into a CUDA graph and replays that graph from then on.
template <class F>
int run_cached(negf_ctx* ctx, int slot, unsigned long long key, bool eligible, F&& body) {
    if (!eligible || !ctx->graph_loops || ctx->prof_on) return body();
    // way with this key, else the least recently used one
    int w = 0;
    for (int q = 0; q < NEGF_GWAYS; q++) if (ctx->gslot[slot][q].key == key) { w = q; goto found; }
    for (int q = 1; q < NEGF_GWAYS; q++) if (ctx->gslot[slot][q].used < ctx->gslot[slot][w].used) w = q;
found:
    negf_ctx::GraphSlot& g = ctx->gslot[slot][w];
    g.used = ++ctx->gtick;
    if (g.exec && g.key == key) {
        NEGF_CUDA_CHECK(ctx, cudaGraphLaunch(g.exec, ctx->stream));
        ctx->launches += g.launches;         // the kernels inside the replayed graph
        return NEGF_OK;
    }
    if (g.key != key) {                      // first sighting: plain run
        if (g.exec) { cudaGraphExecDestroy(g.exec); g.exec = nullptr; }
        g.key = key;
        return body();
    }
    cudaStream_t user = ctx->stream;
    ctx->stream = ctx->cap_stream;
    cudaError_t ce = cudaStreamBeginCapture(ctx->cap_stream, cudaStreamCaptureModeRelaxed);
    if (ce != cudaSuccess) { ctx->stream = user; ctx->last_cuda_error = (int)ce; return NEGF_ECUDA; }
    const long long launches0 = ctx->launches;
    const int rc = body();
    cudaGraph_t G = nullptr;
    ce = cudaStreamEndCapture(ctx->cap_stream, &G);
    ctx->stream = user;
    if (rc != NEGF_OK) { if (G) cudaGraphDestroy(G); return rc; }
    if (ce != cudaSuccess) { ctx->last_cuda_error = (int)ce; return NEGF_ECUDA; }
    ce = cudaGraphInstantiate(&g.exec, G, 0);
    cudaGraphDestroy(G);
    if (ce != cudaSuccess) { g.exec = nullptr; ctx->last_cuda_error = (int)ce; return NEGF_ECUDA; }
    g.launches = ctx->launches - launches0;
    NEGF_CUDA_CHECK(ctx, cudaGraphLaunch(g.exec, ctx->stream));
    return NEGF_OK;
}

// ---- internal entry points (host side, enqueue on ctx->stream) --------------------------------
// zgemm.cu
struct GemmArgs {
    int opA, opB;            // 0 = N, 1 = conjugate transpose
    int m, n, k;
    cplx alpha, beta;
    const cplx* A; int lda; long long sA;
    const cplx* B; int ldb; long long sB;
    const cplx* D; long long sD;   // addend (ld = ldc), may be NULL
    cplx* C; int ldc; long long sC;
    int batch;
    const int* skip;         // optional [batch] device mask: entry skipped when skip[e] != 0
    // optional second batch dimension (the block index i of a family): entry (e, i), e < batch, i < batch2
    int batch2;
    long long sA2, sB2, sD2, sC2;
    const cplx* alpha_vec;   // optional [batch]: entry e uses alpha * alpha_vec[e]
    // C overwrites A in place (C == A, n <= 64): only safe when ONE CTA owns all n columns of its rows, so the
    // launcher must pick a tile with BN >= n (it rejects unflagged aliasing of C with A or B otherwise)
    int c_aliases_a = 0;
};
int zgemm_launch(negf_ctx* ctx, const GemmArgs& a);
int zgemm_prepare(negf_ctx* ctx);
int zinv_prepare(negf_ctx* ctx);      // shared-memory opt-ins of the K1 kernels (zinv.cu)
int econv_prepare(negf_ctx* ctx);     // same for the energy-convolution kernels (econv.cu)
int fused_prepare(negf_ctx* ctx);     // same for the resident small-block kernels (fused_small.cu)
// several independent products of identical shape / ops / batch in ONE launch (blockIdx.z = member)
constexpr int NEGF_GEMM_GROUP_MAX = 4;
// ragged_n: the members may differ in n (and in B, C, D); the grid is laid out for the widest member and the CTAs
// beyond a member's last column tile exit at once (the two rank-w updates of a panel of the blocked inverse)
struct GemmGroup { GemmArgs g[NEGF_GEMM_GROUP_MAX]; int ng; int ragged_n = 0; };
int zgemm_launch_group(negf_ctx* ctx, const GemmGroup& grp);
GemmArgs zgemm_bb_args(int opA, int opB, int b, cplx alpha, const cplx* A, long long sA, const cplx* B, long long sB,
                       cplx beta, const cplx* D, long long sD, cplx* C, long long sC, int batch, const int* skip);
// convenience: square b x b x b, contiguous blocks
int zgemm_bb(negf_ctx* ctx, int opA, int opB, int b, cplx alpha, const cplx* A, long long sA,
             const cplx* B, long long sB, cplx beta, const cplx* D, long long sD,
             cplx* C, long long sC, int batch, const int* skip);

// zinv.cu
size_t zinv_workspace_bytes(int b, int batch);
// in-place inverse of A[e] (b x b, ld = b, stride sA); ws: zinv_workspace_bytes; info_code = value
// written to info[e] on a zero pivot (>0), info untouched otherwise (caller zero-fills).
int zinv_launch(negf_ctx* ctx, int b, cplx* A, long long sA, int batch, void* ws, int* info,
                int info_code, const int* skip, const int* code_dev = nullptr);   // code = *code_dev + info_code (small kernels and the row-per-thread panels)

