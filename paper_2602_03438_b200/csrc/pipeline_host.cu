// The whole S2-S7 path in one call (include/negf.h): negf_pipeline_device (device buffers) and
// negf_pipeline_host (host buffers: what a user without device arrays calls, and what bench.py times as the
// end-to-end number - host->device copies of all inputs, the path, device->host copies of all requested outputs).
//
// K3, the energy-batch scheduler, at the level of the whole path: in the latency-bound small-block regime the
// batch is split into up to four groups of energies that run decimation -> retarded -> lesser/greater ->
// observables concurrently, each on its own stream, child context (side streams, cached graphs) and slice of the
// caller's workspace - one group's inversions overlap another's products.  Forked from and joined to the caller's
// stream inside the call.  Same arithmetic per energy as the four calls; the density is the sum of the groups'
// partial densities in a fixed order.
#include "common.cuh"
#include "workspace.cuh"
#include "fused_small.cuh"

size_t path_workspace_bytes(int n, int b, int ne, bool assembled);

namespace {

struct Bump {
    unsigned char* base; size_t off;
    void* take(size_t bytes) { void* r = base ? base + off : nullptr; off += align_up(bytes, 256); return r; }
};

// energies [lo, lo + cnt) of group g of G
inline void group_range(int ne, int G, int g, int* lo, int* cnt) {
    const int per = (ne + G - 1) / G;
    *lo = min(ne, g * per); *cnt = min(per, ne - *lo);
}

int path_groups(const negf_ctx* ctx, int b, int ne) {
    if (ctx->prof_on) return 1;                     // per-class intervals must not overlap
    int G = ctx->energy_groups;
    if (G == 0 && fused_small_regime(ctx, b, ne)) return 1;       // resident regime: one launch per call covers every energy
    if (G == 0) G = (b <= 96 && ne >= 32) ? NEGF_MAX_ENERGY_GROUPS : 1;
    return max(1, min(min(G, NEGF_MAX_ENERGY_GROUPS), ne));
}

__global__ void merge_info_kernel(int ne, const int* a, const int* b, const int* c, const int* d, int* out) {
    int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= ne) return;
    int v = a[e]; if (!v) v = b[e]; if (!v) v = c[e]; if (!v) v = d[e];
    out[e] = v;
}

// dst[i] = sum_g part[g][i] (partial densities of the energy groups, fixed order)
__global__ void sum_groups_kernel(double* dst, const double* part, int len, int ng) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= len) return;
    double acc = 0.0;
    for (int g = 0; g < ng; g++) acc += part[(size_t)g * len + i];
    dst[i] = acc;
}

// hooks of negf_pipeline_host: device->host copies enqueued per group while the path is still running
struct PathHooks {
    void* user;
    // after negf_rgf_retarded of energies [lo, lo+cnt) has been enqueued on `st`
    int (*after_retarded)(void* user, negf_ctx* ctx, int lo, int cnt, cudaStream_t st, cudaEvent_t ev);
};

int ensure_children(negf_ctx* ctx, int G) {
    if (!ctx->ev_grp_fork) NEGF_CUDA_CHECK(ctx, cudaEventCreateWithFlags(&ctx->ev_grp_fork, cudaEventDisableTiming));
    for (int g = 0; g < G; g++) {
        if (!ctx->child[g]) {
            NEGF_TRY(negf_create(&ctx->child[g], ctx->device));
            NEGF_CUDA_CHECK(ctx, cudaStreamCreateWithFlags(&ctx->grp_stream[g], cudaStreamNonBlocking));
            NEGF_CUDA_CHECK(ctx, cudaEventCreateWithFlags(&ctx->ev_grp_mid[g], cudaEventDisableTiming));
        }
        negf_ctx* c = ctx->child[g];
        c->stream = ctx->grp_stream[g];
        c->graph_loops = ctx->graph_loops; c->gemm_3m = ctx->gemm_3m; c->inv_tensor = ctx->inv_tensor; c->inv_panel = ctx->inv_panel; c->inv_lookahead = ctx->inv_lookahead; c->inv_outer = ctx->inv_outer; c->fused_small = ctx->fused_small;
        // concurrent groups cover each other's launch gaps; a waiting dependent grid would only take their SM slots
        if (c->pdl != 0) negf_set_option(c, NEGF_OPT_PDL, 0);
    }
    return NEGF_OK;
}

inline const void* adv(const void* p, size_t bytes) { return p ? (const char*)p + bytes : nullptr; }
inline void* adv(void* p, size_t bytes) { return p ? (char*)p + bytes : nullptr; }

negf_obc_out slice_obc(const negf_obc_out& o, size_t bb, int lo) {
    negf_obc_out r = o;
    r.sigma_r = (negf_c128*)adv(o.sigma_r, bb * lo); r.gamma = (negf_c128*)adv(o.gamma, bb * lo);
    r.sigma_lesser = (negf_c128*)adv(o.sigma_lesser, bb * lo); r.sigma_greater = (negf_c128*)adv(o.sigma_greater, bb * lo);
    r.g_surface = (negf_c128*)adv(o.g_surface, bb * lo);
    r.fermi = (double*)adv(o.fermi, sizeof(double) * lo);
    r.iters = (int*)adv(o.iters, sizeof(int) * lo); r.status = (int*)adv(o.status, sizeof(int) * lo);
    return r;
}

// the four calls on energies [lo, lo + cnt) of the batch, on context c (its stream, its workspace)
int run_group(negf_ctx* c, const negf_problem* p, const negf_sigma* sig /*[3]*/, bool want_g, const double* weights,
              double mu_L, double mu_R, double kT, double tol, int max_iter, const negf_device_outputs* out,
              int lo, int cnt, double* density_dst, const PathHooks* hooks, cudaEvent_t ev_mid) {
    const int n = p->n_blocks, b = p->block_size, m = n > 1 ? n - 1 : 0;
    const size_t bb = (size_t)b * b * sizeof(cplx), fam_n = bb * n, fam_m = bb * m;
    negf_problem gp = *p;
    gp.n_energy = cnt; gp.energy = p->energy + lo;
    if (p->n_k > 1 && p->k_index) gp.k_index = p->k_index + lo;
    negf_sigma gs[3];
    for (int f = 0; f < 3; f++) {
        gs[f] = sig[f];
        gs[f].scalar = (const negf_c128*)adv(sig[f].scalar, sizeof(cplx) * lo);
        gs[f].diag = (const negf_c128*)adv(sig[f].diag, fam_n * lo);
        gs[f].upper = (const negf_c128*)adv(sig[f].upper, fam_m * lo);
        gs[f].lower = (const negf_c128*)adv(sig[f].lower, fam_m * lo);
    }
    const negf_obc_out oL = slice_obc(out->left, bb, lo), oR = slice_obc(out->right, bb, lo);
    NEGF_TRY(negf_obc_decimate_pair(c, &gp, nullptr, nullptr, mu_L, mu_R, kT, tol, max_iter, &oL, &oR));
    gs[0].left = oL.sigma_r; gs[0].right = oR.sigma_r;
    gs[1].left = oL.sigma_lesser; gs[1].right = oR.sigma_lesser;
    gs[2].left = oL.sigma_greater; gs[2].right = oR.sigma_greater;
    negf_c128* GRd = (negf_c128*)adv(out->GR_diag, fam_n * lo);
    negf_c128* GRu = (negf_c128*)adv(out->GR_upper, fam_m * lo);
    negf_c128* GRl = (negf_c128*)adv(out->GR_lower, fam_m * lo);
    negf_c128* cor = (negf_c128*)adv(out->GR_corner, bb * lo);
    negf_c128* GLd = (negf_c128*)adv(out->GL_diag, fam_n * lo);
    negf_c128* GLu = (negf_c128*)adv(out->GL_upper, fam_m * lo);
    negf_c128* GGd = (negf_c128*)adv(out->GG_diag, fam_n * lo);
    negf_c128* GGu = (negf_c128*)adv(out->GG_upper, fam_m * lo);
    NEGF_TRY(negf_rgf_retarded(c, &gp, &gs[0], GRd, GRu, GRl, cor, NEGF_KEEP_SWEEP, out->info_r + lo));
    if (hooks && hooks->after_retarded) NEGF_TRY(hooks->after_retarded(hooks->user, c, lo, cnt, c->stream, ev_mid));
    NEGF_TRY(negf_rgf_lesser_greater(c, &gp, &gs[0], &gs[1], want_g ? &gs[2] : nullptr, GRd, GLd, GLu, GGd, GGu,
                                     out->info_x + lo));
    const bool mw = want_g && out->contact_current;
    NEGF_TRY(negf_observables(c, &gp, GRd, GRu, GRl, cor, GLd, GLu, GGd, oL.gamma, oR.gamma,
                              mw ? oL.sigma_lesser : nullptr, mw ? oL.sigma_greater : nullptr,
                              mw ? oR.sigma_lesser : nullptr, mw ? oR.sigma_greater : nullptr,
                              weights + lo, density_dst, out->ldos ? out->ldos + (size_t)lo * n : nullptr,
                              (out->transmission && cor) ? out->transmission + lo : nullptr,
                              (out->bond_current && m > 0 && GLu) ? out->bond_current + (size_t)lo * m : nullptr,
                              mw ? out->contact_current + (size_t)lo * 2 : nullptr));
    return NEGF_OK;
}

int run_path(negf_ctx* ctx, const negf_problem* p, const negf_sigma* sr, const negf_sigma* sl, const negf_sigma* sg,
             const double* weights, double mu_L, double mu_R, double kT, double tol, int max_iter,
             const negf_device_outputs* out, const PathHooks* hooks) {
    if (!ctx || !p || !out || !weights) return NEGF_EINVAL;
    const int n = p->n_blocks, b = p->block_size, ne = p->n_energy;
    if (n < 2 || b < 1 || ne < 1 || !p->H_diag || !p->H_upper || !p->energy) return NEGF_EINVAL;   // leads need two blocks (R2)
    if ((p->S_diag == nullptr) != (p->S_upper == nullptr)) return NEGF_EINVAL;
    if (p->n_k > 1 && !p->k_index) return NEGF_EINVAL;
    const bool want_g = sg != nullptr;
    for (const negf_obc_out* o : {&out->left, &out->right})
        if (!o->sigma_r || !o->gamma || !o->sigma_lesser || !o->sigma_greater || !o->iters || !o->status) return NEGF_EINVAL;
    if (!out->GR_diag || !out->GL_diag || !out->info_r || !out->info_x || (want_g && !out->GG_diag)) return NEGF_EINVAL;
    if (!ctx->ws) return NEGF_ENOWORKSPACE;
    negf_sigma sig[3];
    const negf_sigma* in[3] = {sr, sl, sg};
    for (int f = 0; f < 3; f++) { sig[f] = in[f] ? *in[f] : negf_sigma{}; sig[f].left = sig[f].right = nullptr; }
    const bool assembled = p->S_diag != nullptr || sig[0].kind == NEGF_SIGMA_BT || p->n_k > 1;
    const int G = path_groups(ctx, b, ne);
    if (G == 1)
        return run_group(ctx, p, sig, want_g, weights, mu_L, mu_R, kT, tol, max_iter, out, 0, ne, out->density, hooks,
                         ctx->ev_grp[1]);
    // slices of the caller's workspace: one carve-up per group, then the partial densities
    size_t off[NEGF_MAX_ENERGY_GROUPS + 1], total = 0;
    for (int g = 0; g < G; g++) {
        int lo, cnt; group_range(ne, G, g, &lo, &cnt);
        off[g] = total;
        total += align_up(carve_workspace(nullptr, n, b, max(cnt, 1), assembled).bytes, 256);
    }
    off[G] = total;
    const size_t nb = (size_t)n * b;
    if (out->density) total += align_up(sizeof(double) * nb * G, 256);
    if (total > ctx->ws_bytes) return NEGF_ENOWORKSPACE;
    double* part = out->density ? (double*)((char*)ctx->ws + off[G]) : nullptr;
    NEGF_TRY(ensure_children(ctx, G));
    // the regime is a property of the WHOLE batch: a group of a batch that is too large for the resident kernels must
    // not pick them because its own share would fit (b = 32, 296 energies as 4 groups of 74: 7.1 ms against 6.1 ms)
    for (int g = 0; g < G; g++) ctx->child[g]->fused_small = fused_small_regime(ctx, b, ne) ? 2 : 0;
    ctx->sweep_valid = false;                                    // the slices overlay any retained sweep state
    NEGF_CUDA_CHECK(ctx, cudaEventRecord(ctx->ev_grp_fork, ctx->stream));
    int rc = NEGF_OK, used = 0;
    for (int g = 0; g < G && rc == NEGF_OK; g++) {
        int lo, cnt; group_range(ne, G, g, &lo, &cnt);
        if (cnt <= 0) break;
        negf_ctx* c = ctx->child[g];
        const long long l0 = c->launches;
        NEGF_CUDA_CHECK(ctx, cudaStreamWaitEvent(c->stream, ctx->ev_grp_fork, 0));
        void* slice = (char*)ctx->ws + off[g];
        if (c->ws != slice || c->ws_bytes != off[g + 1] - off[g]) negf_set_workspace(c, slice, off[g + 1] - off[g]);
        rc = run_group(c, p, sig, want_g, weights, mu_L, mu_R, kT, tol, max_iter, out, lo, cnt,
                       part ? part + (size_t)g * nb : nullptr, hooks, ctx->ev_grp_mid[g]);
        if (rc == NEGF_ECUDA) ctx->last_cuda_error = c->last_cuda_error;
        ctx->launches += c->launches - l0;
        used = g + 1;
    }
    // join every group that was started, also on failure (nothing of the caller's may be overtaken)
    for (int g = 0; g < used; g++) {
        cudaEventRecord(ctx->ev_grp[g], ctx->child[g]->stream);
        cudaStreamWaitEvent(ctx->stream, ctx->ev_grp[g], 0);
    }
    if (rc != NEGF_OK) return rc;
    if (part) {
        sum_groups_kernel<<<(unsigned)((nb + 255) / 256), 256, 0, ctx->stream>>>(out->density, part, (int)nb, used);
        NEGF_LAUNCH_CHECK(ctx);
    }
    return NEGF_OK;
}

// ---- staging layout of negf_pipeline_host ------------------------------------------------------
struct Layout {
    cplx *Hd, *Hu, *Sd, *Su; double *energy, *weights; int* kidx;
    cplx *sig[3][4];                 // [r,l,g][scalar, diag, upper, lower]
    cplx *ob[2][4];                  // [side][sigma_r, gamma, sl, sg]
    int *iters[2], *status[2];
    cplx *GRd, *GRu, *GRl, *corner, *GLd, *GLu, *GGd, *GGu;
    double *density, *ldos, *trans, *bond, *contact;
    int *info_r, *info_x;
    void* ws; size_t ws_bytes;
    size_t total;
};

// kinds[f] = kind of Sigma^{R,<,>}_S (each family gets the buffers of its OWN kind)
Layout make_layout(void* base, int n, int b, int ne, const int* kinds, bool hasS, bool want_greater, int nk) {
    Layout L = {};
    Bump B{(unsigned char*)base, 0};
    const size_t bb = (size_t)b * b * sizeof(cplx);
    const int m = n > 1 ? n - 1 : 0;
    L.Hd = (cplx*)B.take(bb * n * nk); L.Hu = (cplx*)B.take(bb * m * nk);
    if (hasS) { L.Sd = (cplx*)B.take(bb * n * nk); L.Su = (cplx*)B.take(bb * m * nk); }
    L.energy = (double*)B.take(sizeof(double) * ne); L.weights = (double*)B.take(sizeof(double) * ne);
    if (nk > 1) L.kidx = (int*)B.take(sizeof(int) * ne);
    for (int f = 0; f < 3; f++) {
        if (kinds[f] == NEGF_SIGMA_SCALAR) L.sig[f][0] = (cplx*)B.take(sizeof(cplx) * ne);
        if (kinds[f] == NEGF_SIGMA_BT) {
            L.sig[f][1] = (cplx*)B.take(bb * n * ne); L.sig[f][2] = (cplx*)B.take(bb * m * ne);
            if (f == 0) L.sig[f][3] = (cplx*)B.take(bb * m * ne);
        }
    }
    for (int s = 0; s < 2; s++) {
        for (int k = 0; k < 4; k++) L.ob[s][k] = (cplx*)B.take(bb * ne);
        L.iters[s] = (int*)B.take(sizeof(int) * ne); L.status[s] = (int*)B.take(sizeof(int) * ne);
    }
    L.GRd = (cplx*)B.take(bb * n * ne); L.GRu = (cplx*)B.take(bb * m * ne); L.GRl = (cplx*)B.take(bb * m * ne);
    L.corner = (cplx*)B.take(bb * ne);
    L.GLd = (cplx*)B.take(bb * n * ne); L.GLu = (cplx*)B.take(bb * m * ne);
    if (want_greater) { L.GGd = (cplx*)B.take(bb * n * ne); L.GGu = (cplx*)B.take(bb * m * ne); }
    L.density = (double*)B.take(sizeof(double) * n * b); L.ldos = (double*)B.take(sizeof(double) * ne * n);
    L.trans = (double*)B.take(sizeof(double) * ne); L.bond = (double*)B.take(sizeof(double) * ne * (m > 0 ? m : 1));
    L.contact = (double*)B.take(sizeof(double) * ne * 2);
    L.info_r = (int*)B.take(sizeof(int) * ne); L.info_x = (int*)B.take(sizeof(int) * ne);
    L.ws_bytes = path_workspace_bytes(n, b, ne, hasS || kinds[0] == NEGF_SIGMA_BT || nk > 1);
    L.ws = B.take(L.ws_bytes);
    L.total = B.off;
    return L;
}

struct HostCopies {                      // state of the device->host copies of negf_pipeline_host
    const Layout* L; const negf_host_outputs* out; cudaStream_t cs; size_t down; int n, b;
};

int host_after_retarded(void* user, negf_ctx* c, int lo, int cnt, cudaStream_t st, cudaEvent_t ev) {
    HostCopies* H = (HostCopies*)user;
    const size_t bb = (size_t)H->b * H->b * sizeof(cplx), fam_n = bb * H->n, fam_m = bb * (H->n - 1);
    // G^R of this group goes home on the copy stream while its G^<> is computed
    NEGF_CUDA_CHECK(c, cudaEventRecord(ev, st));
    NEGF_CUDA_CHECK(c, cudaStreamWaitEvent(H->cs, ev, 0));
    struct { void* h; const void* d; size_t per; } cp[3] = {{H->out->GR_diag, H->L->GRd, fam_n}, {H->out->GR_upper, H->L->GRu, fam_m},
                                                            {H->out->GR_lower, H->L->GRl, fam_m}};
    for (auto& q : cp) {
        if (!q.h || !q.per) continue;
        NEGF_CUDA_CHECK(c, cudaMemcpyAsync((char*)q.h + q.per * lo, (const char*)q.d + q.per * lo, q.per * cnt,
                                           cudaMemcpyDeviceToHost, H->cs));
        H->down += q.per * cnt;
    }
    return NEGF_OK;
}

}  // namespace

// workspace that serves every call on this shape, the grouped pipeline included
size_t path_workspace_bytes(int n, int b, int ne, bool assembled) {
    size_t best = carve_workspace(nullptr, n, b, ne, assembled).bytes;
    for (int G = 2; G <= NEGF_MAX_ENERGY_GROUPS && G <= ne; G++) {
        size_t total = 0;
        for (int g = 0; g < G; g++) {
            int lo, cnt; group_range(ne, G, g, &lo, &cnt);
            total += align_up(carve_workspace(nullptr, n, b, max(cnt, 1), assembled).bytes, 256);
        }
        total += align_up(sizeof(double) * (size_t)n * b * G, 256);
        if (total > best) best = total;
    }
    return best;
}

extern "C" int negf_pipeline_device(negf_ctx* ctx, const negf_problem* p, const negf_sigma* sigma_r,
                                    const negf_sigma* sigma_lesser, const negf_sigma* sigma_greater,
                                    const double* weights, double mu_L, double mu_R, double kT, double tol,
                                    int max_iter, const negf_device_outputs* out) {
    return run_path(ctx, p, sigma_r, sigma_lesser, sigma_greater, weights, mu_L, mu_R, kT, tol, max_iter, out, nullptr);
}

extern "C" int negf_pipeline_host_bytes(const negf_problem* p, int kind_max, int want_greater, size_t* bytes) {
    if (!p || !bytes || p->n_blocks < 1 || p->block_size < 1 || p->n_energy < 1) return NEGF_EINVAL;
    const int kinds[3] = {kind_max, kind_max, kind_max};      // an upper bound for any mix of kinds up to kind_max
    Layout L = make_layout(nullptr, p->n_blocks, p->block_size, p->n_energy, kinds, true, want_greater != 0,
                           p->n_k > 1 ? p->n_k : 1);
    *bytes = L.total;
    return NEGF_OK;
}

extern "C" int negf_pipeline_host(negf_ctx* ctx, const negf_problem* hp, const negf_sigma* hsr,
                                  const negf_sigma* hsl, const negf_sigma* hsg, const double* hweights,
                                  double mu_L, double mu_R, double kT, double tol, int max_iter,
                                  void* dev_scratch, size_t dev_scratch_bytes, const negf_host_outputs* out,
                                  size_t* h2d_bytes, size_t* d2h_bytes) {
    if (!ctx || !hp || !out || !dev_scratch || !hweights) return NEGF_EINVAL;
    const int n = hp->n_blocks, b = hp->block_size, ne = hp->n_energy;
    if (n < 2 || b < 1 || ne < 1 || !hp->H_diag || !hp->H_upper || !hp->energy) return NEGF_EINVAL;
    const bool hasS = hp->S_diag != nullptr;
    if (hasS && !hp->S_upper) return NEGF_EINVAL;
    const bool want_g = hsg != nullptr;
    int kinds[3] = {NEGF_SIGMA_NONE, NEGF_SIGMA_NONE, NEGF_SIGMA_NONE};
    const negf_sigma* hs[3] = {hsr, hsl, hsg};
    for (int f = 0; f < 3; f++) {
        if (!hs[f]) continue;
        kinds[f] = hs[f]->kind;
        if (kinds[f] < NEGF_SIGMA_NONE || kinds[f] > NEGF_SIGMA_BT) return NEGF_EINVAL;
        if (kinds[f] == NEGF_SIGMA_SCALAR && !hs[f]->scalar) return NEGF_EINVAL;
        if (kinds[f] == NEGF_SIGMA_BT && (!hs[f]->diag || !hs[f]->upper || (f == 0 && !hs[f]->lower))) return NEGF_EINVAL;
    }
    const int nk = hp->n_k > 1 ? hp->n_k : 1;
    if (nk > 1 && !hp->k_index) return NEGF_EINVAL;
    Layout L = make_layout(dev_scratch, n, b, ne, kinds, hasS, want_g, nk);
    if (L.total > dev_scratch_bytes) return NEGF_ENOWORKSPACE;
    const size_t bb = (size_t)b * b * sizeof(cplx);
    const int m = n - 1;
    size_t up = 0;
    cudaStream_t st = ctx->stream;
    auto H2D = [&](void* d, const void* h, size_t bytes) -> cudaError_t {
        up += bytes; return cudaMemcpyAsync(d, h, bytes, cudaMemcpyHostToDevice, st);
    };
    NEGF_CUDA_CHECK(ctx, H2D(L.Hd, hp->H_diag, bb * n * nk));
    NEGF_CUDA_CHECK(ctx, H2D(L.Hu, hp->H_upper, bb * m * nk));
    if (hasS) {
        NEGF_CUDA_CHECK(ctx, H2D(L.Sd, hp->S_diag, bb * n * nk));
        NEGF_CUDA_CHECK(ctx, H2D(L.Su, hp->S_upper, bb * m * nk));
    }
    if (nk > 1) NEGF_CUDA_CHECK(ctx, H2D(L.kidx, hp->k_index, sizeof(int) * ne));     // HOST k_index here
    NEGF_CUDA_CHECK(ctx, H2D(L.energy, hp->energy, sizeof(double) * ne));
    NEGF_CUDA_CHECK(ctx, H2D(L.weights, hweights, sizeof(double) * ne));
    negf_sigma ds[3];
    for (int f = 0; f < 3; f++) {
        ds[f] = negf_sigma{};
        if (!hs[f]) continue;
        ds[f].kind = hs[f]->kind;
        if (hs[f]->kind == NEGF_SIGMA_SCALAR) {
            NEGF_CUDA_CHECK(ctx, H2D(L.sig[f][0], hs[f]->scalar, sizeof(cplx) * ne));
            ds[f].scalar = (negf_c128*)L.sig[f][0];
        } else if (hs[f]->kind == NEGF_SIGMA_BT) {
            NEGF_CUDA_CHECK(ctx, H2D(L.sig[f][1], hs[f]->diag, bb * n * ne));
            NEGF_CUDA_CHECK(ctx, H2D(L.sig[f][2], hs[f]->upper, bb * m * ne));
            ds[f].diag = (negf_c128*)L.sig[f][1]; ds[f].upper = (negf_c128*)L.sig[f][2];
            if (f == 0) {
                NEGF_CUDA_CHECK(ctx, H2D(L.sig[f][3], hs[f]->lower, bb * m * ne));
                ds[f].lower = (negf_c128*)L.sig[f][3];
            }
        }
    }
    negf_problem dp = *hp;
    dp.H_diag = (negf_c128*)L.Hd; dp.H_upper = (negf_c128*)L.Hu;
    dp.S_diag = hasS ? (negf_c128*)L.Sd : nullptr; dp.S_upper = hasS ? (negf_c128*)L.Su : nullptr;
    dp.energy = L.energy; dp.k_index = nk > 1 ? L.kidx : nullptr;
    negf_device_outputs dout = {};
    negf_obc_out* ob[2] = {&dout.left, &dout.right};
    for (int sd = 0; sd < 2; sd++)
        *ob[sd] = negf_obc_out{(negf_c128*)L.ob[sd][0], (negf_c128*)L.ob[sd][1], (negf_c128*)L.ob[sd][2],
                               (negf_c128*)L.ob[sd][3], nullptr, nullptr, L.iters[sd], L.status[sd]};
    dout.GR_diag = (negf_c128*)L.GRd; dout.GR_upper = (negf_c128*)L.GRu; dout.GR_lower = (negf_c128*)L.GRl;
    dout.GR_corner = (negf_c128*)L.corner; dout.GL_diag = (negf_c128*)L.GLd; dout.GL_upper = (negf_c128*)L.GLu;
    dout.GG_diag = (negf_c128*)L.GGd; dout.GG_upper = (negf_c128*)L.GGu;
    dout.density = out->density ? L.density : nullptr; dout.ldos = out->ldos ? L.ldos : nullptr;
    dout.transmission = out->transmission ? L.trans : nullptr; dout.bond_current = out->bond_current ? L.bond : nullptr;
    dout.contact_current = (out->contact_current && want_g) ? L.contact : nullptr;
    dout.info_r = L.info_r; dout.info_x = L.info_x;

    // the path runs on the staging workspace; the caller's workspace comes back on EVERY exit path, after the
    // copy stream has drained (it reads the staging buffers)
    struct WsGuard {
        negf_ctx* c; void* ws; size_t bytes;
        ~WsGuard() { cudaStreamSynchronize(c->copy_stream); c->ws = ws; c->ws_bytes = bytes; c->sweep_valid = false; }
    } ws_guard{ctx, ctx->ws, ctx->ws_bytes};
    ctx->ws = L.ws; ctx->ws_bytes = L.ws_bytes; ctx->sweep_valid = false;
    cudaStream_t cs = ctx->copy_stream;
    HostCopies H{&L, out, cs, 0, n, b};
    PathHooks hooks{&H, host_after_retarded};
    int rc = run_path(ctx, &dp, &ds[0], &ds[1], want_g ? &ds[2] : nullptr, L.weights, mu_L, mu_R, kT, tol, max_iter,
                      &dout, &hooks);
    if (rc) { cudaStreamSynchronize(st); return rc; }
    size_t down = H.down;
    auto D2H = [&](void* h, const void* d, size_t bytes, cudaStream_t s) -> cudaError_t {
        if (!h || !bytes) return cudaSuccess;
        down += bytes; return cudaMemcpyAsync(h, d, bytes, cudaMemcpyDeviceToHost, s);
    };
    if (out->info) {
        merge_info_kernel<<<(ne + 255) / 256, 256, 0, st>>>(ne, L.status[0], L.status[1], L.info_r, L.info_x, L.info_x);
        NEGF_LAUNCH_CHECK(ctx);
    }
    // the rest of the blocks on the copy stream, the small arrays on the caller's stream
    NEGF_CUDA_CHECK(ctx, cudaEventRecord(ctx->ev_grp[0], st));
    NEGF_CUDA_CHECK(ctx, cudaStreamWaitEvent(cs, ctx->ev_grp[0], 0));
    NEGF_CUDA_CHECK(ctx, D2H(out->GL_diag, L.GLd, bb * n * ne, cs));
    NEGF_CUDA_CHECK(ctx, D2H(out->GL_upper, L.GLu, bb * m * ne, cs));
    if (want_g) {
        NEGF_CUDA_CHECK(ctx, D2H(out->GG_diag, L.GGd, bb * n * ne, cs));
        NEGF_CUDA_CHECK(ctx, D2H(out->GG_upper, L.GGu, bb * m * ne, cs));
    }
    NEGF_CUDA_CHECK(ctx, D2H(out->density, L.density, sizeof(double) * n * b, st));
    NEGF_CUDA_CHECK(ctx, D2H(out->ldos, L.ldos, sizeof(double) * ne * n, st));
    NEGF_CUDA_CHECK(ctx, D2H(out->transmission, L.trans, sizeof(double) * ne, st));
    NEGF_CUDA_CHECK(ctx, D2H(out->bond_current, L.bond, sizeof(double) * ne * m, st));
    if (want_g) NEGF_CUDA_CHECK(ctx, D2H(out->contact_current, L.contact, sizeof(double) * ne * 2, st));
    NEGF_CUDA_CHECK(ctx, D2H(out->info, L.info_x, sizeof(int) * ne, st));
    NEGF_CUDA_CHECK(ctx, cudaStreamSynchronize(st));
    NEGF_CUDA_CHECK(ctx, cudaStreamSynchronize(cs));
    if (h2d_bytes) *h2d_bytes = up;
    if (d2h_bytes) *d2h_bytes = down;
    return NEGF_OK;
}
