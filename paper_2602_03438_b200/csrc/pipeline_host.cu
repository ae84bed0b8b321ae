// negf_pipeline_host: the whole S1-S7 path with HOST buffers (include/negf.h) - what a user
// without device arrays calls, and what bench.py times as the end-to-end number: host->device
// copies of all inputs, the four device calls, device->host copies of all requested outputs.
#include "common.cuh"
#include "workspace.cuh"

namespace {

struct Bump {
    unsigned char* base; size_t off;
    void* take(size_t bytes) { void* r = base ? base + off : nullptr; off += align_up(bytes, 256); return r; }
};

struct Layout {
    cplx *Hd, *Hu, *Sd, *Su; double *energy, *weights;
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
Layout make_layout(void* base, int n, int b, int ne, const int* kinds, bool hasS, bool want_greater) {
    Layout L = {};
    Bump B{(unsigned char*)base, 0};
    const size_t bb = (size_t)b * b * sizeof(cplx);
    const int m = n > 1 ? n - 1 : 0;
    L.Hd = (cplx*)B.take(bb * n); L.Hu = (cplx*)B.take(bb * m);
    if (hasS) { L.Sd = (cplx*)B.take(bb * n); L.Su = (cplx*)B.take(bb * m); }
    L.energy = (double*)B.take(sizeof(double) * ne); L.weights = (double*)B.take(sizeof(double) * ne);
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
    L.density = (double*)B.take(sizeof(double) * n * b * 4); L.ldos = (double*)B.take(sizeof(double) * ne * n);
    L.trans = (double*)B.take(sizeof(double) * ne); L.bond = (double*)B.take(sizeof(double) * ne * (m > 0 ? m : 1));
    L.contact = (double*)B.take(sizeof(double) * ne * 2);
    L.info_r = (int*)B.take(sizeof(int) * ne); L.info_x = (int*)B.take(sizeof(int) * ne);
    Workspace W = carve_workspace(nullptr, n, b, ne, hasS || kinds[0] == NEGF_SIGMA_BT);
    L.ws_bytes = W.bytes; L.ws = B.take(W.bytes);
    L.total = B.off;
    return L;
}

__global__ void merge_info_kernel(int ne, const int* a, const int* b, const int* c, const int* d, int* out) {
    int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= ne) return;
    int v = a[e]; if (!v) v = b[e]; if (!v) v = c[e]; if (!v) v = d[e];
    out[e] = v;
}

// dst[0][i] += dst[g][i], g = 1 .. ng-1 (partial densities of the energy groups)
__global__ void sum_groups_kernel(double* d, int len, int ng) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= len) return;
    double acc = d[i];
    for (int g = 1; g < ng; g++) acc += d[(size_t)g * len + i];
    d[i] = acc;
}

}  // namespace

extern "C" int negf_pipeline_host_bytes(const negf_problem* p, int kind_max, int want_greater, size_t* bytes) {
    if (!p || !bytes || p->n_blocks < 1 || p->block_size < 1 || p->n_energy < 1) return NEGF_EINVAL;
    const int kinds[3] = {kind_max, kind_max, kind_max};      // an upper bound for any mix of kinds up to kind_max
    Layout L = make_layout(nullptr, p->n_blocks, p->block_size, p->n_energy, kinds, true, want_greater != 0);
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
    const bool want_g = hsg != nullptr;
    int kinds[3] = {NEGF_SIGMA_NONE, NEGF_SIGMA_NONE, NEGF_SIGMA_NONE};
    const negf_sigma* hs[3] = {hsr, hsl, hsg};
    for (int f = 0; f < 3; f++) {
        if (!hs[f]) continue;
        kinds[f] = hs[f]->kind;
        if (kinds[f] == NEGF_SIGMA_SCALAR && !hs[f]->scalar) return NEGF_EINVAL;
        if (kinds[f] == NEGF_SIGMA_BT && (!hs[f]->diag || !hs[f]->upper || (f == 0 && !hs[f]->lower))) return NEGF_EINVAL;
        if (kinds[f] < NEGF_SIGMA_NONE || kinds[f] > NEGF_SIGMA_BT) return NEGF_EINVAL;
    }
    Layout L = make_layout(dev_scratch, n, b, ne, kinds, hasS, want_g);
    if (L.total > dev_scratch_bytes) return NEGF_ENOWORKSPACE;
    const size_t bb = (size_t)b * b * sizeof(cplx);
    const int m = n - 1;
    size_t up = 0, down = 0;
    cudaStream_t st = ctx->stream;
    auto H2D = [&](void* d, const void* h, size_t bytes) -> cudaError_t {
        up += bytes; return cudaMemcpyAsync(d, h, bytes, cudaMemcpyHostToDevice, st);
    };
    auto D2H = [&](void* h, const void* d, size_t bytes) -> cudaError_t {
        if (!h) return cudaSuccess;
        down += bytes; return cudaMemcpyAsync(h, d, bytes, cudaMemcpyDeviceToHost, st);
    };
    NEGF_CUDA_CHECK(ctx, H2D(L.Hd, hp->H_diag, bb * n));
    NEGF_CUDA_CHECK(ctx, H2D(L.Hu, hp->H_upper, bb * m));
    if (hasS) {
        if (!hp->S_upper) return NEGF_EINVAL;
        NEGF_CUDA_CHECK(ctx, H2D(L.Sd, hp->S_diag, bb * n));
        NEGF_CUDA_CHECK(ctx, H2D(L.Su, hp->S_upper, bb * m));
    }
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
    dp.energy = L.energy;

    // the four calls below run on the staging workspace; the caller's workspace comes back on EVERY exit path,
    // after the copy stream has drained (it reads the staging buffers)
    struct WsGuard {
        negf_ctx* c; void* ws; size_t bytes;
        ~WsGuard() { cudaStreamSynchronize(c->copy_stream); c->ws = ws; c->ws_bytes = bytes; c->sweep_valid = false; }
    } ws_guard{ctx, ctx->ws, ctx->ws_bytes};
    ctx->ws = L.ws; ctx->ws_bytes = L.ws_bytes; ctx->sweep_valid = false;
    // The device->host copies run on the copy stream and overlap the compute that follows them: G^R goes
    // home while G^<> is computed.  (Splitting the batch into energy groups to overlap more was measured
    // and rejected: the small-block path is bound by its chain latency, which every group pays again.)
    const int G = 1;
    const int per = (ne + G - 1) / G;
    const size_t fam_n = bb * n, fam_m = bb * m;
    cudaStream_t cs = ctx->copy_stream;
    auto D2Hc = [&](void* h, const void* d, size_t bytes) -> cudaError_t {
        if (!h || !bytes) return cudaSuccess;
        down += bytes; return cudaMemcpyAsync(h, d, bytes, cudaMemcpyDeviceToHost, cs);
    };
    auto off = [](const void* p, size_t bytes) -> void* { return p ? (char*)p + bytes : nullptr; };
    int rc = NEGF_OK, ng = 0;
    for (int lo = 0; lo < ne && rc == NEGF_OK; lo += per, ng++) {
        const int cnt = min(per, ne - lo);
        negf_problem gp = dp;
        gp.n_energy = cnt; gp.energy = L.energy + lo;
        negf_sigma gs[3];
        for (int f = 0; f < 3; f++) {
            gs[f] = ds[f];
            gs[f].scalar = (negf_c128*)off(ds[f].scalar, sizeof(cplx) * lo);
            gs[f].diag = (negf_c128*)off(ds[f].diag, fam_n * lo);
            gs[f].upper = (negf_c128*)off(ds[f].upper, fam_m * lo);
            gs[f].lower = (negf_c128*)off(ds[f].lower, fam_m * lo);
        }
        cplx* ob[2][4];
        for (int sd = 0; sd < 2; sd++) for (int k = 0; k < 4; k++) ob[sd][k] = (cplx*)off(L.ob[sd][k], bb * lo);
        negf_obc_out oo[2];
        for (int sd = 0; sd < 2; sd++)
            oo[sd] = negf_obc_out{(negf_c128*)ob[sd][0], (negf_c128*)ob[sd][1], (negf_c128*)ob[sd][2], (negf_c128*)ob[sd][3],
                                  nullptr, nullptr, L.iters[sd] + lo, L.status[sd] + lo};
        rc = negf_obc_decimate_pair(ctx, &gp, nullptr, nullptr, mu_L, mu_R, kT, tol, max_iter, &oo[0], &oo[1]);
        if (rc) break;
        gs[0].left = (negf_c128*)ob[0][0]; gs[0].right = (negf_c128*)ob[1][0];
        gs[1].left = (negf_c128*)ob[0][2]; gs[1].right = (negf_c128*)ob[1][2];
        gs[2].left = (negf_c128*)ob[0][3]; gs[2].right = (negf_c128*)ob[1][3];
        cplx *GRd = (cplx*)off(L.GRd, fam_n * lo), *GRu = (cplx*)off(L.GRu, fam_m * lo), *GRl = (cplx*)off(L.GRl, fam_m * lo);
        cplx *cor = (cplx*)off(L.corner, bb * lo), *GLd = (cplx*)off(L.GLd, fam_n * lo), *GLu = (cplx*)off(L.GLu, fam_m * lo);
        cplx *GGd = (cplx*)off(L.GGd, fam_n * lo), *GGu = (cplx*)off(L.GGu, fam_m * lo);
        rc = negf_rgf_retarded(ctx, &gp, &gs[0], (negf_c128*)GRd, (negf_c128*)GRu, (negf_c128*)GRl, (negf_c128*)cor,
                               NEGF_KEEP_SWEEP, L.info_r + lo);
        if (rc) break;
        NEGF_CUDA_CHECK(ctx, cudaEventRecord(ctx->ev_grp[1], st));
        NEGF_CUDA_CHECK(ctx, cudaStreamWaitEvent(cs, ctx->ev_grp[1], 0));
        NEGF_CUDA_CHECK(ctx, D2Hc(off(out->GR_diag, fam_n * lo), GRd, fam_n * cnt));
        NEGF_CUDA_CHECK(ctx, D2Hc(off(out->GR_upper, fam_m * lo), GRu, fam_m * cnt));
        NEGF_CUDA_CHECK(ctx, D2Hc(off(out->GR_lower, fam_m * lo), GRl, fam_m * cnt));
        rc = negf_rgf_lesser_greater(ctx, &gp, &gs[0], &gs[1], want_g ? &gs[2] : nullptr, (negf_c128*)GRd,
                                     (negf_c128*)GLd, (negf_c128*)GLu, (negf_c128*)GGd, (negf_c128*)GGu, L.info_x + lo);
        if (rc) break;
        double* dens = out->density ? L.density + (size_t)ng * n * b : nullptr;      // partial density of this group
        rc = negf_observables(ctx, &gp, (negf_c128*)GRd, (negf_c128*)GRu, (negf_c128*)GRl, (negf_c128*)cor,
                              (negf_c128*)GLd, (negf_c128*)GLu, (negf_c128*)GGd,
                              (negf_c128*)ob[0][1], (negf_c128*)ob[1][1],
                              (negf_c128*)ob[0][2], (negf_c128*)ob[0][3], (negf_c128*)ob[1][2], (negf_c128*)ob[1][3],
                              L.weights + lo, dens, out->ldos ? L.ldos + (size_t)lo * n : nullptr,
                              out->transmission ? L.trans + lo : nullptr, out->bond_current ? L.bond + (size_t)lo * m : nullptr,
                              (out->contact_current && want_g) ? L.contact + (size_t)lo * 2 : nullptr);
        if (rc) break;
        if (out->info) {
            merge_info_kernel<<<(cnt + 255) / 256, 256, 0, st>>>(cnt, L.status[0] + lo, L.status[1] + lo, L.info_r + lo,
                                                                L.info_x + lo, L.info_x + lo);
            NEGF_LAUNCH_CHECK(ctx);
        }
        // this group's results go home on the copy stream
        NEGF_CUDA_CHECK(ctx, cudaEventRecord(ctx->ev_grp[ng], st));
        NEGF_CUDA_CHECK(ctx, cudaStreamWaitEvent(cs, ctx->ev_grp[ng], 0));
        NEGF_CUDA_CHECK(ctx, D2Hc(off(out->GL_diag, fam_n * lo), GLd, fam_n * cnt));
        NEGF_CUDA_CHECK(ctx, D2Hc(off(out->GL_upper, fam_m * lo), GLu, fam_m * cnt));
        if (want_g) {
            NEGF_CUDA_CHECK(ctx, D2Hc(off(out->GG_diag, fam_n * lo), GGd, fam_n * cnt));
            NEGF_CUDA_CHECK(ctx, D2Hc(off(out->GG_upper, fam_m * lo), GGu, fam_m * cnt));
        }
    }
    if (rc) { cudaStreamSynchronize(st); return rc; }
    if (out->density) {          // total density = sum of the groups' partial densities, fixed order
        sum_groups_kernel<<<(n * b + 255) / 256, 256, 0, st>>>(L.density, n * b, ng);
        NEGF_LAUNCH_CHECK(ctx);
    }
    NEGF_CUDA_CHECK(ctx, D2H(out->density, L.density, sizeof(double) * n * b));
    NEGF_CUDA_CHECK(ctx, D2H(out->ldos, L.ldos, sizeof(double) * ne * n));
    NEGF_CUDA_CHECK(ctx, D2H(out->transmission, L.trans, sizeof(double) * ne));
    NEGF_CUDA_CHECK(ctx, D2H(out->bond_current, L.bond, sizeof(double) * ne * m));
    if (want_g) NEGF_CUDA_CHECK(ctx, D2H(out->contact_current, L.contact, sizeof(double) * ne * 2));
    NEGF_CUDA_CHECK(ctx, D2H(out->info, L.info_x, sizeof(int) * ne));
    NEGF_CUDA_CHECK(ctx, cudaStreamSynchronize(st));
    NEGF_CUDA_CHECK(ctx, cudaStreamSynchronize(cs));
    if (h2d_bytes) *h2d_bytes = up;
    if (d2h_bytes) *d2h_bytes = down;
    return NEGF_OK;
}
