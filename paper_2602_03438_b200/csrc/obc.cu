// S2: open-boundary self-energies by Sancho-Rubio doubling, all energies
// in lock-step.  The paper only says an "open boundary condition term" enters B;
// the algorithm is the one BASELINE.json:north_star names.  Energies that met the stopping rule
// (reading R3) are masked out of every later launch through the device-side `done` flags, so the
// host enqueues max_iter doublings without ever synchronising.
#include "common.cuh"
#include "kernels.cuh"
#include "workspace.cuh"

extern "C" int negf_obc_decimate(negf_ctx* ctx, const negf_problem* p, const negf_lead* lead, int side,
                                 double mu, double kT, double tol, int max_iter,
                                 negf_c128* sigma_r, negf_c128* gamma, negf_c128* sigma_lesser,
                                 negf_c128* sigma_greater, negf_c128* g_surface, double* fermi,
                                 int* iters, int* status) {
    if (!ctx || !p || !sigma_r || !iters || !status) return NEGF_EINVAL;
    if (side != 0 && side != 1) return NEGF_EINVAL;
    const int n = p->n_blocks, b = p->block_size, ne = p->n_energy;
    if (n < 1 || b < 1 || ne < 1 || max_iter < 1 || !p->energy) return NEGF_EINVAL;
    if ((p->S_diag == nullptr) != (p->S_upper == nullptr) && n > 1) return NEGF_EINVAL;
    const cplx *Hd, *Hu, *Sd, *Su;
    const size_t bb = (size_t)b * b;
    if (lead) {
        Hd = (const cplx*)lead->H_d; Hu = (const cplx*)lead->H_u;
        Sd = (const cplx*)lead->S_d; Su = (const cplx*)lead->S_u;
        if (!Hd || !Hu) return NEGF_EINVAL;
    } else {
        if (n < 2 || !p->H_diag || !p->H_upper) return NEGF_EINVAL;   // periodic copies need two blocks (R2)
        const cplx* HD = (const cplx*)p->H_diag; const cplx* HU = (const cplx*)p->H_upper;
        const cplx* SD = (const cplx*)p->S_diag; const cplx* SU = (const cplx*)p->S_upper;
        if (side == 0) { Hd = HD; Hu = HU; Sd = SD; Su = SU; }
        else {
            Hd = HD + bb * (n - 1); Hu = HU + bb * (n - 2);
            Sd = SD ? SD + bb * (n - 1) : nullptr; Su = SU ? SU + bb * (n - 2) : nullptr;
        }
    }
    if (!ctx->ws) return NEGF_ENOWORKSPACE;
    Workspace W = carve_workspace(ctx->ws, n, b, ne);
    if (W.bytes > ctx->ws_bytes) return NEGF_ENOWORKSPACE;

    cplx *a_s = W.T[0], *a_b = W.T[1], *U0 = W.T[2], *L0 = W.T[3];
    cplx *ub[2] = {W.T[4], W.T[6]}, *lb[2] = {W.T[5], W.T[7]};
    cplx *g = W.T[8], *gu = W.T[9], *gl = W.T[10], *lgu = W.T[11], *ugl = W.T[12];
    const long long sb = (long long)bb;
    const cplx one = cmake(1.0, 0.0), mone = cmake(-1.0, 0.0), zero = cmake(0.0, 0.0);

    // lead blocks a_d, a_u, a_l for every energy
    CombineArgs ca = {};
    ca.b = b; ca.energy = p->energy; ca.eta = p->eta; ca.use_z = 1; ca.coef = -1.0; ca.sout = sb; ca.skip = nullptr;
    ca.H = Hd; ca.S = Sd; ca.s_identity = Sd ? 0 : 1; ca.dagger = 0; ca.out = a_s;
    NEGF_TRY(ew_combine(ctx, ca, ne));
    NEGF_TRY(ew_copy(ctx, bb, ne, a_b, sb, a_s, sb, nullptr));
    ca.H = Hu; ca.S = Su; ca.s_identity = 0; ca.dagger = 0; ca.out = U0;
    NEGF_TRY(ew_combine(ctx, ca, ne));
    ca.dagger = 1; ca.out = L0;
    NEGF_TRY(ew_combine(ctx, ca, ne));
    NEGF_TRY(ew_fill_int(ctx, W.done, ne, 0));
    NEGF_TRY(ew_fill_int(ctx, W.sing, ne, 0));
    NEGF_TRY(ew_fill_int(ctx, iters, ne, 0));
    NEGF_TRY(ew_sr_norm(ctx, b, ne, U0, L0, W.ref, tol, W.done, iters, 0, 0));

    const cplx* u = U0; const cplx* l = L0;
    for (int it = 0; it < max_iter; it++) {
        const int* skip = W.done;
        cplx* un = ub[it & 1]; cplx* ln = lb[it & 1];
        NEGF_TRY(ew_copy(ctx, bb, ne, g, sb, a_b, sb, skip));
        NEGF_TRY(zinv_launch(ctx, b, g, sb, ne, W.inv, W.sing, it + 1, skip));
        NEGF_TRY(zgemm_bb(ctx, 0, 0, b, one, g, sb, u, sb, zero, nullptr, 0, gu, sb, ne, skip));     // g u
        NEGF_TRY(zgemm_bb(ctx, 0, 0, b, one, g, sb, l, sb, zero, nullptr, 0, gl, sb, ne, skip));     // g l
        NEGF_TRY(zgemm_bb(ctx, 0, 0, b, one, l, sb, gu, sb, zero, nullptr, 0, lgu, sb, ne, skip));   // l g u
        NEGF_TRY(zgemm_bb(ctx, 0, 0, b, one, u, sb, gl, sb, zero, nullptr, 0, ugl, sb, ne, skip));   // u g l
        NEGF_TRY(ew_sr_update(ctx, b, ne, side, a_s, a_b, lgu, ugl, skip));
        NEGF_TRY(zgemm_bb(ctx, 0, 0, b, mone, u, sb, gu, sb, zero, nullptr, 0, un, sb, ne, skip));   // u <- -u g u
        NEGF_TRY(zgemm_bb(ctx, 0, 0, b, mone, l, sb, gl, sb, zero, nullptr, 0, ln, sb, ne, skip));   // l <- -l g l
        NEGF_TRY(ew_sr_norm(ctx, b, ne, un, ln, W.ref, tol, W.done, iters, it, 1));
        // a converged energy keeps its last (u, l) in whichever buffer; they are not used again
        u = un; l = ln;
    }
    // g_s = a_s^-1 ; Sigma = a_l g_s a_u (left) | a_u g_s a_l (right)
    NEGF_TRY(zinv_launch(ctx, b, a_s, sb, ne, W.inv, W.sing, max_iter + 1, nullptr));
    if (g_surface) NEGF_TRY(ew_copy(ctx, bb, ne, (cplx*)g_surface, sb, a_s, sb, nullptr));
    const cplx* first = side == 0 ? L0 : U0;
    const cplx* last = side == 0 ? U0 : L0;
    NEGF_TRY(zgemm_bb(ctx, 0, 0, b, one, a_s, sb, last, sb, zero, nullptr, 0, gu, sb, ne, nullptr));
    NEGF_TRY(zgemm_bb(ctx, 0, 0, b, one, first, sb, gu, sb, zero, nullptr, 0, (cplx*)sigma_r, sb, ne, nullptr));
    NEGF_TRY(ew_obc_finalize(ctx, b, ne, (const cplx*)sigma_r, p->energy, mu, kT, (cplx*)gamma,
                             (cplx*)sigma_lesser, (cplx*)sigma_greater, fermi));
    NEGF_TRY(ew_obc_status(ctx, ne, W.done, W.sing, status));
    return NEGF_OK;
}
