// S2: open-boundary self-energies by Sancho-Rubio doubling, all energies
// in lock-step.  The paper only says an "open boundary condition term" enters B;
// the algorithm is the one BASELINE.json:north_star names.  Energies that met the stopping rule
// (reading R3) are masked out of every later launch through the device-side `done` flags, so the
// host enqueues max_iter doublings without ever synchronising.
//
// Scheduling (K3): a right lead is the left-lead recursion with the roles of u and l exchanged
// (a_s -= u g l, Sigma = a_u g_s a_l), so both leads of all energies run as ONE batch of 2 N_E
// uniform entries when the blocks are small (b <= NEGF_PAIR_MAX_B); the two / four independent
// products of a doubling share one grouped GEMM launch, and for small blocks the update, the
// norms and the convergence test are one kernel: 4 launches per doubling.
#include "common.cuh"
#include "kernels.cuh"
#include "workspace.cuh"
#include "fused_small.cuh"
#include "zinv_rows.cuh"

namespace {

struct LeadBlocks { const cplx *Hd, *Hu, *Sd, *Su; long long kd, ku; };   // kd / ku: strides between k-points

int resolve_lead(const negf_problem* p, const negf_lead* lead, int side, LeadBlocks* out) {
    const int n = p->n_blocks;
    const size_t bb = (size_t)p->block_size * p->block_size;
    if (lead) {
        out->Hd = (const cplx*)lead->H_d; out->Hu = (const cplx*)lead->H_u;
        out->Sd = (const cplx*)lead->S_d; out->Su = (const cplx*)lead->S_u;
        out->kd = out->ku = (long long)bb;
        return (out->Hd && out->Hu) ? NEGF_OK : NEGF_EINVAL;
    }
    if (n < 2 || !p->H_diag || !p->H_upper) return NEGF_EINVAL;   // periodic copies need two blocks (R2)
    const cplx* HD = (const cplx*)p->H_diag; const cplx* HU = (const cplx*)p->H_upper;
    const cplx* SD = (const cplx*)p->S_diag; const cplx* SU = (const cplx*)p->S_upper;
    out->kd = (long long)bb * n; out->ku = (long long)bb * (n - 1);
    if (side == 0) { out->Hd = HD; out->Hu = HU; out->Sd = SD; out->Su = SU; }
    else {
        out->Hd = HD + bb * (n - 1); out->Hu = HU + bb * (n - 2);
        out->Sd = SD ? SD + bb * (n - 1) : nullptr; out->Su = SU ? SU + bb * (n - 2) : nullptr;
    }
    return NEGF_OK;
}

// ns = 1 or 2 leads stacked in the batch dimension: entry s*ne + e.
int obc_core(negf_ctx* ctx, const negf_problem* p, int ns, const LeadBlocks* lb, const int* sides, const double* mus,
             double kT, double tol, int max_iter, const negf_obc_out* const* outs) {
    const int n = p->n_blocks, b = p->block_size, ne = p->n_energy, nb = ns * ne;
    const size_t bb = (size_t)b * b;
    const long long sb = (long long)bb;
    if (fused_small_regime(ctx, b, ne)) {
        // resident small-block regime: one CTA per (lead, energy) walks the whole doubling loop (fused_small.cu)
        FusedObcArgs fa = {};
        fa.b = b; fa.ne = ne; fa.ns = ns; fa.energy = p->energy; fa.eta = p->eta;
        fa.kidx = p->n_k > 1 ? p->k_index : nullptr; fa.kT = kT; fa.tol = tol; fa.max_iter = max_iter;
        for (int s = 0; s < ns; s++) {
            const negf_obc_out* o = outs[s];
            fa.lead[s] = FusedLead{lb[s].Hd, lb[s].Hu, lb[s].Sd, lb[s].Su, lb[s].kd, lb[s].ku, sides[s], mus[s],
                                   (cplx*)o->sigma_r, (cplx*)o->gamma, (cplx*)o->sigma_lesser, (cplx*)o->sigma_greater,
                                   (cplx*)o->g_surface, o->fermi, o->iters, o->status};
        }
        return fused_obc_launch(ctx, fa);
    }
    Workspace W = carve_workspace(ctx->ws, n, b, ne);
    if (W.bytes > ctx->ws_bytes) return NEGF_ENOWORKSPACE;
    cplx *a_s = W.T[0], *a_b = W.T[1], *U0 = W.T[2], *L0 = W.T[3];
    cplx *ub[2] = {W.T[4], W.T[6]}, *lbuf[2] = {W.T[5], W.T[7]};
    cplx *g = W.T[8], *gu = W.T[9], *gl = W.T[10], *lgu = W.T[11], *ugl = W.T[12];
    const cplx one = cmake(1.0, 0.0), mone = cmake(-1.0, 0.0), zero = cmake(0.0, 0.0);

    // lead blocks a_d, a_u, a_l for every energy; a right lead stores (u, l) exchanged
    for (int s = 0; s < ns; s++) {
        const size_t off = (size_t)s * ne * bb;
        CombineArgs ca = {};
        ca.b = b; ca.energy = p->energy; ca.eta = p->eta; ca.use_z = 1; ca.coef = -1.0; ca.sout = sb; ca.skip = nullptr;
        ca.kidx = p->n_k > 1 ? p->k_index : nullptr;
        ca.H = lb[s].Hd; ca.S = lb[s].Sd; ca.s_identity = lb[s].Sd ? 0 : 1; ca.dagger = 0; ca.out = a_s + off;
        ca.kH = ca.kS = lb[s].kd;
        NEGF_TRY(ew_combine(ctx, ca, ne));
        ca.H = lb[s].Hu; ca.S = lb[s].Su; ca.s_identity = 0; ca.kH = ca.kS = lb[s].ku;
        ca.dagger = 0; ca.out = (sides[s] == 0 ? U0 : L0) + off;      // a_u
        NEGF_TRY(ew_combine(ctx, ca, ne));
        ca.dagger = 1; ca.out = (sides[s] == 0 ? L0 : U0) + off;      // a_l
        NEGF_TRY(ew_combine(ctx, ca, ne));
    }
    NEGF_TRY(ew_copy(ctx, bb, nb, a_b, sb, a_s, sb, nullptr));
    NEGF_TRY(ew_copy(ctx, bb, nb, g, sb, a_s, sb, nullptr));
    NEGF_TRY(ew_fill_int(ctx, W.done, nb, 0));
    NEGF_TRY(ew_fill_int(ctx, W.sing, nb, 0));
    NEGF_TRY(ew_fill_int(ctx, W.its, nb, 0));
    NEGF_CUDA_CHECK(ctx, cudaMemsetAsync(W.ticket, 0, sizeof(unsigned) * nb, ctx->stream));
    NEGF_TRY(ew_sr_norm(ctx, b, nb, U0, L0, W.ref, tol, W.done, W.its, 0, 0));

    const bool fused_step = true;      // update + norms + stopping rule in one kernel at every block size
    // one doubling: reads (u, l), writes (un, ln); `it` is the host iteration index, or the offset
    // added to the device counter it_dev inside the WHILE graph
    auto doubling = [&](const cplx* u, const cplx* l, cplx* un, cplx* ln, int it, const int* it_dev) -> int {
        const int* skip = W.done;
        NEGF_TRY(zinv_launch(ctx, b, g, sb, nb, W.inv, W.sing, it + 1, skip, it_dev));     // g = a_b^-1
        GemmGroup g1; g1.ng = 2;
        g1.g[0] = zgemm_bb_args(0, 0, b, one, g, sb, u, sb, zero, nullptr, 0, gu, sb, nb, skip);    // g u
        g1.g[1] = zgemm_bb_args(0, 0, b, one, g, sb, l, sb, zero, nullptr, 0, gl, sb, nb, skip);    // g l
        NEGF_TRY(zgemm_launch_group(ctx, g1));
        GemmGroup g2; g2.ng = 4;
        g2.g[0] = zgemm_bb_args(0, 0, b, one, l, sb, gu, sb, zero, nullptr, 0, lgu, sb, nb, skip);  // l g u
        g2.g[1] = zgemm_bb_args(0, 0, b, one, u, sb, gl, sb, zero, nullptr, 0, ugl, sb, nb, skip);  // u g l
        g2.g[2] = zgemm_bb_args(0, 0, b, mone, u, sb, gu, sb, zero, nullptr, 0, un, sb, nb, skip);  // u <- -u g u
        g2.g[3] = zgemm_bb_args(0, 0, b, mone, l, sb, gl, sb, zero, nullptr, 0, ln, sb, nb, skip);  // l <- -l g l
        NEGF_TRY(zgemm_launch_group(ctx, g2));
        if (fused_step) {
            NEGF_TRY(ew_sr_step(ctx, b, nb, a_s, a_b, g, lgu, ugl, un, ln, W.ref, tol, W.done, W.its, it, W.acc, W.ticket, it_dev));
        } else {
            NEGF_TRY(ew_sr_update(ctx, b, nb, a_s, a_b, g, lgu, ugl, skip));
            NEGF_TRY(ew_sr_norm(ctx, b, nb, un, ln, W.ref, tol, W.done, W.its, it, 1));
        }
        return NEGF_OK;
    };
    // Small blocks: the loop is a device-driven WHILE graph (CUDA conditional node): its body is two
    // doublings (so the ping-pong buffers have fixed roles) plus a kernel that keeps the loop going
    // while any entry is active - no masked launches after convergence, no host synchronisation.
    // The graph is cached per (workspace, n, b, N_E, leads in the batch, tol, max_iter) - everything the baked-in
    // workspace offsets depend on - and dropped by negf_set_workspace; profiling runs use the plain loop.
    // Above b = 96 (NEGF_OPT_GRAPH_LOOPS = 2) the body holds the ~300 launches of two blocked inverses with their
    // look-ahead side stream (a fork and join inside the capture); the zero-pivot code of the row-per-thread panels
    // follows the device iteration counter, the first-generation panel kernels have no such argument.
    const bool use_graph = (b <= 96 || (ctx->graph_loops >= 2 && gj_panel_rows_supported(b) && ctx->inv_panel)) &&
                           (max_iter % 2 == 0) && !ctx->prof_on && ctx->graph_loops;
    if (use_graph) {
        int* it_dev = W.tmpinfo;
        NEGF_TRY(ew_copy(ctx, bb, nb, ub[1], sb, U0, sb, nullptr));
        NEGF_TRY(ew_copy(ctx, bb, nb, lbuf[1], sb, L0, sb, nullptr));
        NEGF_TRY(ew_fill_int(ctx, it_dev, 1, 0));
        const bool hit = ctx->obc_exec && ctx->obc_key_ws == ctx->ws && ctx->obc_key_b == b && ctx->obc_key_n == n &&
                         ctx->obc_key_ne == ne && ctx->obc_key_ns == ns &&
                         ctx->obc_key_maxit == max_iter && ctx->obc_key_tol == tol;
        if (!hit) {
            if (ctx->obc_exec) { cudaGraphExecDestroy(ctx->obc_exec); ctx->obc_exec = nullptr; }
            cudaGraph_t G = nullptr;
            NEGF_CUDA_CHECK(ctx, cudaGraphCreate(&G, 0));
            cudaGraphConditionalHandle h;
            NEGF_CUDA_CHECK(ctx, cudaGraphConditionalHandleCreate(&h, G, 1, cudaGraphCondAssignDefault));
            cudaGraphNodeParams np = {};
            np.type = cudaGraphNodeTypeConditional;
            np.conditional.handle = h; np.conditional.type = cudaGraphCondTypeWhile; np.conditional.size = 1;
            cudaGraphNode_t node;
            NEGF_CUDA_CHECK(ctx, cudaGraphAddNode(&node, G, nullptr, 0, &np));
            cudaGraph_t body = np.conditional.phGraph_out[0];
            // captured on a side stream: the caller's stream may be the legacy default stream, which cannot capture
            StreamFork sf(ctx);
            sf.use_side(0);
            cudaError_t ce = cudaStreamBeginCaptureToGraph(ctx->stream, body, nullptr, nullptr, 0, cudaStreamCaptureModeRelaxed);
            if (ce != cudaSuccess) { cudaGraphDestroy(G); ctx->last_cuda_error = (int)ce; return NEGF_ECUDA; }
            int rc = NEGF_OK;
            const long long launches0 = ctx->launches;
            ctx->in_while_body = true;
            const int dpb = 2;         // doublings per WHILE iteration (4 / 8 measured: 5.77 / 5.74 ms against 5.79 at configs[1])
            for (int q = 0; q < dpb && rc == NEGF_OK; q += 2) {
                rc = doubling(ub[1], lbuf[1], ub[0], lbuf[0], q, it_dev);
                if (rc == NEGF_OK) rc = doubling(ub[0], lbuf[0], ub[1], lbuf[1], q + 1, it_dev);
            }
            if (rc == NEGF_OK) rc = ew_sr_cond(ctx, h, nb, W.done, it_dev, max_iter, dpb);
            cudaGraph_t dummy = nullptr;
            ce = cudaStreamEndCapture(ctx->stream, &dummy);
            ctx->in_while_body = false;
            sf.use_main();
            if (rc != NEGF_OK) { cudaGraphDestroy(G); return rc; }
            if (ce != cudaSuccess) { cudaGraphDestroy(G); ctx->last_cuda_error = (int)ce; return NEGF_ECUDA; }
            ce = cudaGraphInstantiate(&ctx->obc_exec, G, 0);
            cudaGraphDestroy(G);
            if (ce != cudaSuccess) { ctx->obc_exec = nullptr; ctx->last_cuda_error = (int)ce; return NEGF_ECUDA; }
            ctx->obc_body_launches = ctx->launches - launches0;
            ctx->obc_key_ws = ctx->ws; ctx->obc_key_b = b; ctx->obc_key_n = n; ctx->obc_key_ne = ne; ctx->obc_key_ns = ns; ctx->obc_key_maxit = max_iter; ctx->obc_key_tol = tol;
        }
        NEGF_CUDA_CHECK(ctx, cudaGraphLaunch(ctx->obc_exec, ctx->stream));
    } else {
        const cplx* u = U0; const cplx* l = L0;
        for (int it = 0; it < max_iter; it++) {
            cplx* un = ub[it & 1]; cplx* ln = lbuf[it & 1];
            NEGF_TRY(doubling(u, l, un, ln, it, nullptr));
            // a converged entry keeps its last (u, l) in whichever buffer; they are not used again
            u = un; l = ln;
        }
    }
    // g_s = a_s^-1 ; Sigma = a_l g_s a_u (in the exchanged storage of a right lead: a_u g_s a_l)
    NEGF_TRY(zinv_launch(ctx, b, a_s, sb, nb, W.inv, W.sing, max_iter + 1, nullptr));
    NEGF_TRY(zgemm_bb(ctx, 0, 0, b, one, a_s, sb, U0, sb, zero, nullptr, 0, gu, sb, nb, nullptr));
    GemmGroup gs; gs.ng = ns;
    for (int s = 0; s < ns; s++) {
        const size_t off = (size_t)s * ne * bb;
        gs.g[s] = zgemm_bb_args(0, 0, b, one, L0 + off, sb, gu + off, sb, zero, nullptr, 0, (cplx*)outs[s]->sigma_r, sb, ne, nullptr);
    }
    NEGF_TRY(zgemm_launch_group(ctx, gs));
    for (int s = 0; s < ns; s++) {
        const negf_obc_out* o = outs[s];
        const size_t off = (size_t)s * ne * bb;
        if (o->g_surface) NEGF_TRY(ew_copy(ctx, bb, ne, (cplx*)o->g_surface, sb, a_s + off, sb, nullptr));
        NEGF_TRY(ew_obc_finalize(ctx, b, ne, (const cplx*)o->sigma_r, p->energy, mus[s], kT, (cplx*)o->gamma,
                                 (cplx*)o->sigma_lesser, (cplx*)o->sigma_greater, o->fermi));
        NEGF_TRY(ew_obc_status(ctx, ne, W.done + s * ne, W.sing + s * ne, W.its + s * ne, o->status, o->iters));
    }
    return NEGF_OK;
}

int check_common(const negf_ctx* ctx, const negf_problem* p, int max_iter) {
    if (!ctx || !p) return NEGF_EINVAL;
    if (p->n_blocks < 1 || p->block_size < 1 || p->n_energy < 1 || max_iter < 1 || !p->energy) return NEGF_EINVAL;
    if ((p->S_diag == nullptr) != (p->S_upper == nullptr) && p->n_blocks > 1) return NEGF_EINVAL;
    if (p->n_k > 1 && !p->k_index) return NEGF_EINVAL;
    if (!ctx->ws && !fused_small_regime(ctx, p->block_size, p->n_energy)) return NEGF_ENOWORKSPACE;
    return NEGF_OK;
}

}  // namespace

extern "C" int negf_obc_decimate(negf_ctx* ctx, const negf_problem* p, const negf_lead* lead, int side,
                                 double mu, double kT, double tol, int max_iter,
                                 negf_c128* sigma_r, negf_c128* gamma, negf_c128* sigma_lesser,
                                 negf_c128* sigma_greater, negf_c128* g_surface, double* fermi,
                                 int* iters, int* status) {
    if (!sigma_r || !iters || !status) return NEGF_EINVAL;
    if (side != 0 && side != 1) return NEGF_EINVAL;
    NEGF_TRY(check_common(ctx, p, max_iter));
    LeadBlocks lb;
    NEGF_TRY(resolve_lead(p, lead, side, &lb));
    negf_obc_out o = {sigma_r, gamma, sigma_lesser, sigma_greater, g_surface, fermi, iters, status};
    const negf_obc_out* po = &o;
    return obc_core(ctx, p, 1, &lb, &side, &mu, kT, tol, max_iter, &po);
}

extern "C" int negf_obc_decimate_pair(negf_ctx* ctx, const negf_problem* p, const negf_lead* lead_L,
                                      const negf_lead* lead_R, double mu_L, double mu_R, double kT, double tol,
                                      int max_iter, const negf_obc_out* left, const negf_obc_out* right) {
    if (!left || !right || !left->sigma_r || !right->sigma_r || !left->iters || !right->iters ||
        !left->status || !right->status) return NEGF_EINVAL;
    NEGF_TRY(check_common(ctx, p, max_iter));
    LeadBlocks lb[2];
    NEGF_TRY(resolve_lead(p, lead_L, 0, &lb[0]));
    NEGF_TRY(resolve_lead(p, lead_R, 1, &lb[1]));
    const int sides[2] = {0, 1};
    const double mus[2] = {mu_L, mu_R};
    const negf_obc_out* outs[2] = {left, right};
    if (negf_tmul(p->block_size) == 2) return obc_core(ctx, p, 2, lb, sides, mus, kT, tol, max_iter, outs);
    // large blocks fill the machine on their own: one lead after the other, half the scratch
    NEGF_TRY(obc_core(ctx, p, 1, &lb[0], &sides[0], &mus[0], kT, tol, max_iter, &outs[0]));
    return obc_core(ctx, p, 1, &lb[1], &sides[1], &mus[1], kT, tol, max_iter, &outs[1]);
}
