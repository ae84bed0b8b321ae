// S1 + S3-S6: the RGF sweeps, all energies of the batch in lock-step
// ("Each E is independent of the other"; "sequential in essence" along the
// blocks).  K3, the energy-batch scheduler: every sweep step is one batched launch
// of the K2 GEMM / K1 inverse over the energy axis, and everything that does NOT sit on the
// sequential chain is hoisted out of it and batched over (energy x block index) in one launch:
//   S4  X_i = g_i A_{i,i+1} for all i; then two launches per block (grouped Gu / Gl / corner, G_ii);
//   S5  (small blocks or ballistic) g^x_i = W_i + Z_i g^x_{i-1} Z_i^H with W_i = g_i [..] g_i^H and
//       Z_i = g_i A_{i,i-1} batched over i: two launches per block instead of four;
//   S6  T2_i, Q_i = T2_i (G^R_{i+1,i+1})^H and P_i = g^x_i - Q_i X_i^H batched over i; then
//       G^x_{i,i+1} = Q_i - X_i G^x_{i+1,i+1} and G^x_ii = P_i + X_i (G^x_{i,i+1})^H (same five
//       products per block as the textbook form, two on the chain, no elementwise pass).
// S1: with S = I and no block-tridiagonal Sigma^R_S the off-diagonal blocks of A are -H_{i,i+1}
// and its dagger for every energy, so they are read straight from H (operand flags, alpha = -1)
// and never materialised; otherwise the two off-diagonal families are assembled once per call.
// The diagonal blocks are assembled straight into the g family and inverted in place.
#include "rgf_common.cuh"
#include "fused_small.cuh"

using namespace rgfc;

size_t path_workspace_bytes(int n, int b, int ne, bool assembled);   // pipeline_host.cu

extern "C" int negf_workspace_bytes(const negf_problem* p, int kind_max, int flags, size_t* bytes) {
    (void)flags;
    if (!p || !bytes || p->n_blocks < 1 || p->block_size < 1 || p->n_energy < 1) return NEGF_EINVAL;
    const bool assembled = p->S_diag != nullptr || kind_max == NEGF_SIGMA_BT || p->n_k > 1;
    // covers the four calls on the whole batch AND the per-group slices + partial densities of negf_pipeline_device
    *bytes = path_workspace_bytes(p->n_blocks, p->block_size, p->n_energy, assembled);
    return NEGF_OK;
}

// S1: the diagonal blocks of A into the g family (inverted in place later) and, when they depend on
// the energy, the two off-diagonal families.
int rgf_assemble(negf_ctx* ctx, const negf_problem* p, const negf_sigma* sigma_r, const Shape& s, const Workspace& W,
                 bool assembled) {
    const int b = s.b, ne = s.ne, n = s.n;
    // S1: diagonal blocks A_ii = z S_ii - H_ii - Sigma^R_ii for all i straight into the g family
    {
        CombineArgs ca = {};
        ca.b = b; ca.energy = p->energy; ca.eta = p->eta; ca.use_z = 1; ca.coef = -1.0;
        ca.H = (const cplx*)p->H_diag; ca.fH = s.sb;
        ca.S = (const cplx*)p->S_diag; ca.fS = s.sb; ca.s_identity = p->S_diag ? 0 : 1;
        ca.kidx = kidx_of(p); ca.kH = s.sn; ca.kS = s.sn;
        ca.out = W.g; ca.sout = s.sn; ca.fout = s.sb; ca.nfam = n;
        int nb = 0;
        if (sigma_r) {
            if (sigma_r->kind == NEGF_SIGMA_SCALAR) ca.scalar = (const cplx*)sigma_r->scalar;
            if (sigma_r->kind == NEGF_SIGMA_BT) { ca.blk[nb] = (const cplx*)sigma_r->diag; ca.sblk[nb] = s.sn; ca.fblk[nb] = s.sb; ca.only[nb] = -1; nb++; }
            if (sigma_r->left) { ca.blk[nb] = (const cplx*)sigma_r->left; ca.sblk[nb] = s.sb; ca.only[nb] = 0; nb++; }
            if (sigma_r->right) { ca.blk[nb] = (const cplx*)sigma_r->right; ca.sblk[nb] = s.sb; ca.only[nb] = n - 1; nb++; }
        }
        if (n == 1) {   // a single launch slot (blockIdx.z = 0) must take both boundary blocks
            ca.nfam = 1;
        }
        NEGF_TRY(ew_combine(ctx, ca, ne));
    }
    if (assembled && n > 1) {   // off-diagonal families, once per call
        for (int which = 1; which <= 2; which++) {
            CombineArgs ca = {};
            ca.b = b; ca.energy = p->energy; ca.eta = p->eta; ca.use_z = 1; ca.coef = -1.0;
            ca.H = (const cplx*)p->H_upper; ca.fH = s.sb; ca.S = (const cplx*)p->S_upper; ca.fS = s.sb; ca.s_identity = 0;
            ca.kidx = kidx_of(p); ca.kH = s.sm; ca.kS = s.sm;
            ca.dagger = (which == 2);
            ca.out = which == 1 ? W.Aup : W.Alow; ca.sout = s.sm; ca.fout = s.sb; ca.nfam = n - 1;
            if (sigma_r && sigma_r->kind == NEGF_SIGMA_BT) {
                ca.blk[0] = (const cplx*)(which == 1 ? sigma_r->upper : sigma_r->lower);
                ca.sblk[0] = s.sm; ca.fblk[0] = s.sb; ca.only[0] = -1;
            }
            if (n - 1 == 1) ca.nfam = 1;
            NEGF_TRY(ew_combine(ctx, ca, ne));
        }
    }

    return NEGF_OK;
}

namespace {
FusedProblem fused_problem(const negf_problem* p, const negf_sigma* sr) {
    FusedProblem P = {};
    P.n = p->n_blocks; P.b = p->block_size; P.ne = p->n_energy;
    P.Hd = (const cplx*)p->H_diag; P.Hu = (const cplx*)p->H_upper; P.Sd = (const cplx*)p->S_diag; P.Su = (const cplx*)p->S_upper;
    P.energy = p->energy; P.eta = p->eta; P.kidx = kidx_of(p);
    P.sr_kind = sr ? sr->kind : NEGF_SIGMA_NONE;
    if (sr) {
        P.sr_scalar = (const cplx*)sr->scalar; P.sr_diag = (const cplx*)sr->diag; P.sr_upper = (const cplx*)sr->upper;
        P.sr_lower = (const cplx*)sr->lower; P.sr_left = (const cplx*)sr->left; P.sr_right = (const cplx*)sr->right;
    }
    return P;
}
}  // namespace

extern "C" int negf_rgf_retarded(negf_ctx* ctx, const negf_problem* p, const negf_sigma* sigma_r,
                                 negf_c128* GR_diag_, negf_c128* GR_upper_, negf_c128* GR_lower_,
                                 negf_c128* GR_corner_, int flags, int* info) {
    NEGF_TRY(check_problem(ctx, p));
    if (!GR_diag_ || !info) return NEGF_EINVAL;
    const Shape s = shape_of(p);
    NEGF_TRY(check_sigma(sigma_r, s.n, true));
    if (!ctx->ws) return NEGF_ENOWORKSPACE;
    const bool assembled = needs_assembly(p, sigma_r);
    Workspace W = carve_workspace(ctx->ws, s.n, s.b, s.ne, assembled);
    if (W.bytes > ctx->ws_bytes) return NEGF_ENOWORKSPACE;
    ctx->sweep_valid = false;
    const int b = s.b, ne = s.ne, n = s.n;
    const Fams F = make_fams(p, s, W, assembled);
    const Opnd GRd = {(const cplx*)GR_diag_, s.sn, s.sb, 0};
    if (fused_small_regime(ctx, b, ne)) {     // resident regime: one CTA per energy walks both sweeps
        NEGF_TRY(ew_fill_int(ctx, info, ne, 0));
        const FusedProblem P = fused_problem(p, sigma_r);
        const FusedRetOut fo = {W.g, W.X, W.Y, (cplx*)GR_diag_, (cplx*)GR_upper_, (cplx*)GR_lower_, (cplx*)GR_corner_, info};
        NEGF_TRY(fused_ret_launch(ctx, P, fo));
        if (flags & NEGF_KEEP_SWEEP) { ctx->sweep_valid = true; ctx->sw_n = n; ctx->sw_b = b; ctx->sw_ne = ne; ctx->sw_assembled = assembled; ctx->sw_fused = true; }
        return NEGF_OK;
    }
    ctx->sw_fused = false;
    if (b <= NEGF_PAIR_MAX_B) {      // latency-bound regime: two-sided sweeps (rgf2.cu), replayed as a cached graph
        KeyHash k;
        k.val(*p); if (sigma_r) k.val(*sigma_r);
        k.val(GR_diag_); k.val(GR_upper_); k.val(GR_lower_); k.val(GR_corner_); k.val(info); k.val(ctx->ws); k.val(ctx->ws_bytes);
        NEGF_TRY(run_cached(ctx, 0, k.h, b <= 96, [&]() -> int {
            NEGF_TRY(ew_fill_int(ctx, info, ne, 0));
            NEGF_TRY(rgf_assemble(ctx, p, sigma_r, s, W, assembled));
            return rgf2_retarded(ctx, p, s, W, F, (cplx*)GR_diag_, (cplx*)GR_upper_, (cplx*)GR_lower_, (cplx*)GR_corner_, info);
        }));
        if (flags & NEGF_KEEP_SWEEP) { ctx->sweep_valid = true; ctx->sw_n = n; ctx->sw_b = b; ctx->sw_ne = ne; ctx->sw_assembled = assembled; }
        return NEGF_OK;
    }
    NEGF_TRY(ew_fill_int(ctx, info, ne, 0));
    NEGF_TRY(rgf_assemble(ctx, p, sigma_r, s, W, assembled));

    // S3 forward: g_0 = A_00^-1 ; Y_{i-1} = A_{i,i-1} g_{i-1} ; g_i = (A_ii - Y_{i-1} A_{i-1,i})^-1
    for (int i = 0; i < n; i++) {
        if (i > 0) {
            NEGF_TRY(zgemm_launch(ctx, gemm_one(s, real(F.sgn), F.AL, i - 1, F.g, i - 1, ZERO, nullptr, 0, F.Y, i - 1)));
            NEGF_TRY(zgemm_launch(ctx, gemm_one(s, real(-F.sgn), F.Y, i - 1, F.AU, i - 1, ONE, &F.g, i, F.g, i)));
        }
        NEGF_TRY(zinv_launch(ctx, b, W.g + s.bb * i, s.sn, ne, W.inv, info, i + 1, nullptr));
    }
    // S4 backward
    NEGF_TRY(ew_copy(ctx, s.bb, ne, (cplx*)GR_diag_ + s.bb * (n - 1), s.sn, W.g + s.bb * (n - 1), s.sn, nullptr));
    if (n > 1) NEGF_TRY(launch_fam(ctx, s, real(F.sgn), F.g, 0, F.AU, 0, ZERO, nullptr, 0, F.X, 0, n - 1));   // X_i, all i
    cplx* col = W.T[3]; cplx* coln = W.T[5];
    if (GR_corner_) NEGF_TRY(ew_copy(ctx, s.bb, ne, n > 1 ? col : (cplx*)GR_corner_, s.sb, W.g + s.bb * (n - 1), s.sn, nullptr));
    const Opnd GRu = GR_upper_ ? Opnd{(const cplx*)GR_upper_, s.sm, s.sb, 0} : Opnd{W.T[4], s.sb, 0, 0};
    const Opnd GRl = {(const cplx*)GR_lower_, s.sm, s.sb, 0};
    for (int i = n - 2; i >= 0; i--) {
        GemmGroup grp; grp.ng = 0;
        grp.g[grp.ng++] = gemm_one(s, MONE, F.X, i, GRd, i + 1, ZERO, nullptr, 0, GRu, GR_upper_ ? i : 0);   // G_{i,i+1}
        if (GR_lower_) grp.g[grp.ng++] = gemm_one(s, MONE, GRd, i + 1, F.Y, i, ZERO, nullptr, 0, GRl, i);     // G_{i+1,i}
        if (GR_corner_) {                                                                                     // G_{i,n-1}
            cplx* dst = (i == 0) ? (cplx*)GR_corner_ : coln;
            grp.g[grp.ng++] = gemm_one(s, MONE, F.X, i, Opnd{col, s.sb, 0, 0}, 0, ZERO, nullptr, 0, Opnd{dst, s.sb, 0, 0}, 0);
            cplx* t = col; col = coln; coln = t;
        }
        NEGF_TRY(zgemm_launch_group(ctx, grp));
        NEGF_TRY(zgemm_launch(ctx, gemm_one(s, MONE, GRu, GR_upper_ ? i : 0, F.Y, i, ONE, &F.g, i, GRd, i)));  // G_ii
    }
    if (flags & NEGF_KEEP_SWEEP) { ctx->sweep_valid = true; ctx->sw_n = n; ctx->sw_b = b; ctx->sw_ne = ne; ctx->sw_assembled = assembled; }
    return NEGF_OK;
}

namespace {

// B_ii contribution of the boundary blocks at the two ends: gx_i (+)= g_i B g_i^H
int add_boundary_w(negf_ctx* ctx, const Shape& s, const Fams& F, const Workspace& W, const cplx* bnd, int i, bool accumulate) {
    if (!bnd) return NEGF_OK;
    const Opnd Bn = {bnd, s.sb, 0, 0}, T = {W.T[0], s.sb, 0, 0};
    NEGF_TRY(zgemm_launch(ctx, gemm_one(s, ONE, F.g, i, Bn, 0, ZERO, nullptr, 0, T, 0)));
    return zgemm_launch(ctx, gemm_one(s, ONE, T, 0, dag(F.g), i, accumulate ? ONE : ZERO, accumulate ? &F.gx : nullptr, i, F.gx, i));
}

// S5, hoisted form: g^x_i = W_i + Z_i g^x_{i-1} Z_i^H
int s5_hoisted(negf_ctx* ctx, const Shape& s, const Fams& F, const Workspace& W, const negf_sigma* sx) {
    const int n = s.n, ne = s.ne, b = s.b;
    bool have_w = false;     // interior W_i present in the gx family
    if (sx->kind == NEGF_SIGMA_SCALAR) {
        NEGF_TRY(launch_fam(ctx, s, ONE, F.g, 0, dag(F.g), 0, ZERO, nullptr, 0, F.gx, 0, n, (const cplx*)sx->scalar));
        have_w = true;
    } else if (sx->kind == NEGF_SIGMA_BT) {
        const Opnd Sd = {(const cplx*)sx->diag, s.sn, s.sb, 0}, Su = {(const cplx*)sx->upper, s.sm, s.sb, 0};
        // bracket_i = Sigma_ii - (V_i - V_i^H), V_i = Y_{i-1} Sigma_{i-1,i} (i >= 1), built in the gx family
        NEGF_TRY(ew_copy(ctx, s.bb, ne, W.gx, s.sn, Sd.p, s.sn, nullptr));
        if (n > 1) {
            NEGF_TRY(launch_fam(ctx, s, ONE, F.Y, 0, Su, 0, ZERO, nullptr, 0, F.Q, 1, n - 1));
            for (int i = 1; i < n; i++)
                NEGF_TRY(ew_antiherm_add(ctx, b, ne, W.gx + s.bb * i, s.sn, Sd.p + s.bb * i, s.sn, W.Q + s.bb * i, s.sn, -1.0));
        }
        NEGF_TRY(launch_fam(ctx, s, ONE, F.g, 0, F.gx, 0, ZERO, nullptr, 0, F.Q, 0, n));
        NEGF_TRY(launch_fam(ctx, s, ONE, F.Q, 0, dag(F.g), 0, ZERO, nullptr, 0, F.gx, 0, n));
        have_w = true;
    }
    bool first_set = have_w;
    if (sx->left) { NEGF_TRY(add_boundary_w(ctx, s, F, W, (const cplx*)sx->left, 0, first_set)); first_set = true; }
    if (n == 1 && sx->right) { NEGF_TRY(add_boundary_w(ctx, s, F, W, (const cplx*)sx->right, 0, first_set)); first_set = true; }
    if (!first_set)          // g^x_0 = 0
        NEGF_CUDA_CHECK(ctx, cudaMemset2DAsync(W.gx, (size_t)s.sn * sizeof(cplx), 0, s.bb * sizeof(cplx), ne, ctx->stream));
    bool last_has_w = have_w;
    if (n > 1 && sx->right) { NEGF_TRY(add_boundary_w(ctx, s, F, W, (const cplx*)sx->right, n - 1, have_w)); last_has_w = true; }
    if (n == 1) return NEGF_OK;
    NEGF_TRY(launch_fam(ctx, s, real(F.sgn), F.g, 1, F.AL, 0, ZERO, nullptr, 0, F.Z, 0, n - 1));      // Z_i = g_i A_{i,i-1}
    const Opnd T = {W.T[1], s.sb, 0, 0};
    for (int i = 1; i < n; i++) {
        const bool w = (i == n - 1) ? last_has_w : have_w;
        NEGF_TRY(zgemm_launch(ctx, gemm_one(s, ONE, F.Z, i - 1, F.gx, i - 1, ZERO, nullptr, 0, T, 0)));
        NEGF_TRY(zgemm_launch(ctx, gemm_one(s, ONE, T, 0, dag(F.Z), i - 1, w ? ONE : ZERO, w ? &F.gx : nullptr, i, F.gx, i)));
    }
    return NEGF_OK;
}

// S5, textbook form (fewest products when Sigma^x_S is dense): g^x_i = g_i [B_ii + A g^x_{i-1} A^H - (V - V^H)] g_i^H
int s5_textbook(negf_ctx* ctx, const Shape& s, const Fams& F, const Workspace& W, const negf_sigma* sx) {
    const int n = s.n, ne = s.ne, b = s.b;
    const Opnd T0 = {W.T[0], s.sb, 0, 0}, T2 = {W.T[2], s.sb, 0, 0}, T3 = {W.T[3], s.sb, 0, 0}, T5 = {W.T[5], s.sb, 0, 0};
    for (int i = 0; i < n; i++) {
        // B_ii into T0
        CombineArgs ca = {};
        ca.b = b; ca.use_z = 0; ca.coef = 1.0; ca.out = W.T[0]; ca.sout = s.sb;
        int nb = 0;
        if (sx->kind == NEGF_SIGMA_SCALAR) ca.scalar = (const cplx*)sx->scalar;
        if (sx->kind == NEGF_SIGMA_BT) { ca.blk[nb] = (const cplx*)sx->diag + s.bb * i; ca.sblk[nb] = s.sn; nb++; }
        if (i == 0 && sx->left) { ca.blk[nb] = (const cplx*)sx->left; ca.sblk[nb] = s.sb; nb++; }
        if (i == n - 1 && sx->right) { ca.blk[nb] = (const cplx*)sx->right; ca.sblk[nb] = s.sb; nb++; }
        NEGF_TRY(ew_combine(ctx, ca, ne));
        const Opnd* M = &T0;
        if (i > 0) {
            NEGF_TRY(zgemm_launch(ctx, gemm_one(s, real(F.sgn), F.AL, i - 1, F.gx, i - 1, ZERO, nullptr, 0, T2, 0)));
            NEGF_TRY(zgemm_launch(ctx, gemm_one(s, real(F.sgn), T2, 0, dag(F.AL), i - 1, ONE, &T0, 0, T3, 0)));
            if (sx->kind == NEGF_SIGMA_BT) {
                const Opnd Su = {(const cplx*)sx->upper, s.sm, s.sb, 0};
                NEGF_TRY(zgemm_launch(ctx, gemm_one(s, ONE, F.Y, i - 1, Su, i - 1, ZERO, nullptr, 0, T5, 0)));
                NEGF_TRY(ew_antiherm_add(ctx, b, ne, W.T[3], s.sb, W.T[3], s.sb, W.T[5], s.sb, -1.0));
            }
            M = &T3;
        }
        NEGF_TRY(zgemm_launch(ctx, gemm_one(s, ONE, F.g, i, *M, 0, ZERO, nullptr, 0, T2, 0)));
        NEGF_TRY(zgemm_launch(ctx, gemm_one(s, ONE, T2, 0, dag(F.g), i, ZERO, nullptr, 0, F.gx, i)));
    }
    return NEGF_OK;
}

// S5 + S6 for one of </>.  GXd [NE][n][b][b] required, GXu [NE][n-1][b][b] optional.
int lesser_greater_one(negf_ctx* ctx, const negf_problem* p, const negf_sigma* sx, const Shape& s, const Workspace& W,
                       const Fams& F, const cplx* GRd_, cplx* GXd_, cplx* GXu_) {
    (void)p;
    const int ne = s.ne, n = s.n;
    const bool dense_sx = sx->kind != NEGF_SIGMA_NONE;
    if (dense_sx && s.b > NEGF_PAIR_MAX_B) NEGF_TRY(s5_textbook(ctx, s, F, W, sx));
    else NEGF_TRY(s5_hoisted(ctx, s, F, W, sx));
    // S6 backward
    NEGF_TRY(ew_copy(ctx, s.bb, ne, GXd_ + s.bb * (n - 1), s.sn, W.gx + s.bb * (n - 1), s.sn, nullptr));
    if (n == 1) return NEGF_OK;
    const Opnd GRd = {GRd_, s.sn, s.sb, 0}, GXd = {GXd_, s.sn, s.sb, 0};
    const Opnd Qf = GXu_ ? Opnd{GXu_, s.sm, s.sb, 0} : Opnd{W.Q, s.sn, s.sb, 0};
    // T2_i = -g^x_i A_{i+1,i}^H (+ g_i Sigma_{i,i+1}) into the Z family
    NEGF_TRY(launch_fam(ctx, s, real(-F.sgn), F.gx, 0, dag(F.AL), 0, ZERO, nullptr, 0, F.Z, 0, n - 1));
    if (sx->kind == NEGF_SIGMA_BT) {
        const Opnd Su = {(const cplx*)sx->upper, s.sm, s.sb, 0};
        NEGF_TRY(launch_fam(ctx, s, ONE, F.g, 0, Su, 0, ONE, &F.Z, 0, F.Z, 0, n - 1));
    }
    NEGF_TRY(launch_fam(ctx, s, ONE, F.Z, 0, dag(GRd), 1, ZERO, nullptr, 0, Qf, 0, n - 1));          // Q_i
    NEGF_TRY(launch_fam(ctx, s, MONE, Qf, 0, dag(F.X), 0, ONE, &F.gx, 0, GXd, 0, n - 1));            // P_i
    for (int i = n - 2; i >= 0; i--) {
        NEGF_TRY(zgemm_launch(ctx, gemm_one(s, MONE, F.X, i, GXd, i + 1, ONE, &Qf, i, Qf, i)));     // G^x_{i,i+1}
        NEGF_TRY(zgemm_launch(ctx, gemm_one(s, ONE, F.X, i, dag(Qf), i, ONE, &GXd, i, GXd, i)));    // G^x_ii
    }
    return NEGF_OK;
}

}  // namespace

extern "C" int negf_rgf_lesser_greater(negf_ctx* ctx, const negf_problem* p, const negf_sigma* sigma_r,
                                       const negf_sigma* sigma_lesser, const negf_sigma* sigma_greater,
                                       const negf_c128* GR_diag, negf_c128* GL_diag, negf_c128* GL_upper,
                                       negf_c128* GG_diag, negf_c128* GG_upper, int* info) {
    NEGF_TRY(check_problem(ctx, p));
    if (!GR_diag || !info) return NEGF_EINVAL;
    const Shape s = shape_of(p);
    NEGF_TRY(check_sigma(sigma_r, s.n, true));
    NEGF_TRY(check_sigma(sigma_lesser, s.n, false));
    NEGF_TRY(check_sigma(sigma_greater, s.n, false));
    if (sigma_lesser && !GL_diag) return NEGF_EINVAL;
    if (sigma_greater && !GG_diag) return NEGF_EINVAL;
    if (!ctx->ws) return NEGF_ENOWORKSPACE;
    const bool assembled = needs_assembly(p, sigma_r);
    Workspace W = carve_workspace(ctx->ws, s.n, s.b, s.ne, assembled);
    if (W.bytes > ctx->ws_bytes) return NEGF_ENOWORKSPACE;
    if (!ctx->sweep_valid || ctx->sw_n != s.n || ctx->sw_b != s.b || ctx->sw_ne != s.ne || ctx->sw_assembled != assembled)
        return NEGF_ENOSTATE;
    const Fams F = make_fams(p, s, W, assembled);
    if (ctx->sw_fused) {            // state left by the resident small-block kernel: S5 + S6 in one launch, too
        NEGF_TRY(ew_fill_int(ctx, info, s.ne, 0));
        const FusedProblem P = fused_problem(p, sigma_r);
        FusedLgArgs la = {};
        la.g = W.g; la.X = W.X; la.Y = W.Y; la.GR_diag = (const cplx*)GR_diag;
        const negf_sigma* sx[2] = {sigma_lesser, sigma_greater};
        cplx* gxw[2] = {W.gx, W.Q};
        cplx* od[2] = {(cplx*)GL_diag, (cplx*)GG_diag};
        cplx* ou[2] = {(cplx*)GL_upper, (cplx*)GG_upper};
        for (int q = 0; q < 2; q++) {
            if (!sx[q]) continue;
            la.x[la.nx++] = FusedLgOne{sx[q]->kind, (const cplx*)sx[q]->scalar, (const cplx*)sx[q]->diag, (const cplx*)sx[q]->upper,
                                       (const cplx*)sx[q]->left, (const cplx*)sx[q]->right, gxw[q], od[q], ou[q]};
        }
        return la.nx ? fused_lg_launch(ctx, P, la) : NEGF_OK;
    }
    const bool two_sided = s.b <= NEGF_PAIR_MAX_B;
    KeyHash k;
    k.val(*p); if (sigma_r) k.val(*sigma_r); if (sigma_lesser) k.val(*sigma_lesser); if (sigma_greater) k.val(*sigma_greater);
    k.val(sigma_lesser != nullptr); k.val(sigma_greater != nullptr);
    k.val(GR_diag); k.val(GL_diag); k.val(GL_upper); k.val(GG_diag); k.val(GG_upper); k.val(info); k.val(ctx->ws); k.val(ctx->ws_bytes);
    return run_cached(ctx, 1, k.h, two_sided && s.b <= 96, [&]() -> int {
    NEGF_TRY(ew_fill_int(ctx, info, s.ne, 0));
    if (sigma_lesser)
        NEGF_TRY(two_sided ? rgf2_lesser_greater_one(ctx, sigma_lesser, s, W, F, (const cplx*)GR_diag, (cplx*)GL_diag, (cplx*)GL_upper)
                           : lesser_greater_one(ctx, p, sigma_lesser, s, W, F, (const cplx*)GR_diag, (cplx*)GL_diag, (cplx*)GL_upper));
    if (sigma_greater)
        NEGF_TRY(two_sided ? rgf2_lesser_greater_one(ctx, sigma_greater, s, W, F, (const cplx*)GR_diag, (cplx*)GG_diag, (cplx*)GG_upper)
                           : lesser_greater_one(ctx, p, sigma_greater, s, W, F, (const cplx*)GR_diag, (cplx*)GG_diag, (cplx*)GG_upper));
    return NEGF_OK;
    });
}
