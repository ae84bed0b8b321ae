// S1 + S3-S6: the RGF sweeps, all energies of the batch in lock-step
// ("Each E is independent of the other"; "sequential in essence" along the
// blocks).  Every sweep step is one batched launch of the K2 GEMM / K1 inverse
// over the energy axis (K3: the energy-batch scheduler for the large-block regime).
// The blocks of A = z S - H - Sigma^R are assembled per step into scratch and never stored as
// a family (S1).
#include "common.cuh"
#include "kernels.cuh"
#include "workspace.cuh"

namespace {

struct Shape { int n, b, ne; size_t bb; long long sb, sn, sm; };   // sn = n*bb, sm = (n-1)*bb

Shape shape_of(const negf_problem* p) {
    Shape s;
    s.n = p->n_blocks; s.b = p->block_size; s.ne = p->n_energy;
    s.bb = (size_t)s.b * s.b; s.sb = (long long)s.bb; s.sn = (long long)s.bb * s.n;
    s.sm = (long long)s.bb * (s.n - 1);
    return s;
}

int check_problem(const negf_ctx* ctx, const negf_problem* p) {
    if (!ctx || !p) return NEGF_EINVAL;
    if (p->n_blocks < 1 || p->block_size < 1 || p->n_energy < 1) return NEGF_EINVAL;
    if (!p->H_diag || !p->energy) return NEGF_EINVAL;
    if (p->n_blocks > 1 && !p->H_upper) return NEGF_EINVAL;
    if (p->n_blocks > 1 && ((p->S_diag == nullptr) != (p->S_upper == nullptr))) return NEGF_EINVAL;
    if (p->n_energy > 65535) return NEGF_EUNSUPPORTED;
    return NEGF_OK;
}

int check_sigma(const negf_sigma* s, int n, bool retarded) {
    if (!s) return NEGF_OK;
    if (s->kind == NEGF_SIGMA_NONE) return NEGF_OK;
    if (s->kind == NEGF_SIGMA_SCALAR) return s->scalar ? NEGF_OK : NEGF_EINVAL;
    if (s->kind == NEGF_SIGMA_BT) {
        if (!s->diag) return NEGF_EINVAL;
        if (n > 1 && !s->upper) return NEGF_EINVAL;
        if (n > 1 && retarded && !s->lower) return NEGF_EINVAL;
        return NEGF_OK;
    }
    return NEGF_EINVAL;
}

// A-block `which` (0 diag i, 1 upper i = A_{i,i+1}, 2 lower i = A_{i+1,i}) for all energies.
int assemble_a(negf_ctx* ctx, const negf_problem* p, const negf_sigma* sr, const Shape& s, int which,
               int i, cplx* out, long long sout) {
    CombineArgs ca = {};
    ca.b = s.b; ca.energy = p->energy; ca.eta = p->eta; ca.use_z = 1; ca.coef = -1.0;
    ca.out = out; ca.sout = sout; ca.skip = nullptr;
    const cplx* HD = (const cplx*)p->H_diag; const cplx* HU = (const cplx*)p->H_upper;
    const cplx* SD = (const cplx*)p->S_diag; const cplx* SU = (const cplx*)p->S_upper;
    int nb = 0;
    if (which == 0) {
        ca.H = HD + s.bb * i; ca.S = SD ? SD + s.bb * i : nullptr; ca.s_identity = SD ? 0 : 1; ca.dagger = 0;
        if (sr) {
            if (sr->kind == NEGF_SIGMA_SCALAR) ca.scalar = (const cplx*)sr->scalar;
            if (sr->kind == NEGF_SIGMA_BT) { ca.blk[nb] = (const cplx*)sr->diag + s.bb * i; ca.sblk[nb] = s.sn; nb++; }
            if (i == 0 && sr->left) { ca.blk[nb] = (const cplx*)sr->left; ca.sblk[nb] = s.sb; nb++; }
            if (i == s.n - 1 && sr->right) { ca.blk[nb] = (const cplx*)sr->right; ca.sblk[nb] = s.sb; nb++; }
        }
    } else {
        ca.H = HU + s.bb * i; ca.S = SU ? SU + s.bb * i : nullptr; ca.s_identity = 0; ca.dagger = (which == 2);
        if (sr && sr->kind == NEGF_SIGMA_BT) {
            ca.blk[0] = (const cplx*)(which == 1 ? sr->upper : sr->lower) + s.bb * i; ca.sblk[0] = s.sm;
        }
    }
    return ew_combine(ctx, ca, s.ne);
}

// B-block of Sigma^x: which 0 = diag i, 1 = upper i.  *is_zero set when nothing contributes.
int assemble_b(negf_ctx* ctx, const negf_sigma* sx, const Shape& s, int which, int i, cplx* out,
               bool* is_zero) {
    CombineArgs ca = {};
    ca.b = s.b; ca.use_z = 0; ca.coef = 1.0; ca.out = out; ca.sout = s.sb; ca.skip = nullptr;
    int nb = 0; bool any = false;
    if (which == 0) {
        if (sx->kind == NEGF_SIGMA_SCALAR) { ca.scalar = (const cplx*)sx->scalar; any = true; }
        if (sx->kind == NEGF_SIGMA_BT) { ca.blk[nb] = (const cplx*)sx->diag + s.bb * i; ca.sblk[nb] = s.sn; nb++; }
        if (i == 0 && sx->left) { ca.blk[nb] = (const cplx*)sx->left; ca.sblk[nb] = s.sb; nb++; }
        if (i == s.n - 1 && sx->right) { ca.blk[nb] = (const cplx*)sx->right; ca.sblk[nb] = s.sb; nb++; }
    } else {
        if (sx->kind == NEGF_SIGMA_BT) { ca.blk[nb] = (const cplx*)sx->upper + s.bb * i; ca.sblk[nb] = s.sm; nb++; }
    }
    any = any || nb > 0;
    *is_zero = !any;
    if (!any && which == 1) return NEGF_OK;     // callers skip the products with a zero upper block
    return ew_combine(ctx, ca, s.ne);
}

const cplx ONE = {1.0, 0.0}, MONE = {-1.0, 0.0}, ZERO = {0.0, 0.0};

}  // namespace

extern "C" int negf_workspace_bytes(const negf_problem* p, int kind_max, int flags, size_t* bytes) {
    (void)kind_max; (void)flags;
    if (!p || !bytes || p->n_blocks < 1 || p->block_size < 1 || p->n_energy < 1) return NEGF_EINVAL;
    Workspace w = carve_workspace(nullptr, p->n_blocks, p->block_size, p->n_energy);
    *bytes = w.bytes;
    return NEGF_OK;
}

extern "C" int negf_rgf_retarded(negf_ctx* ctx, const negf_problem* p, const negf_sigma* sigma_r,
                                 negf_c128* GR_diag_, negf_c128* GR_upper_, negf_c128* GR_lower_,
                                 negf_c128* GR_corner_, int flags, int* info) {
    NEGF_TRY(check_problem(ctx, p));
    if (!GR_diag_ || !info) return NEGF_EINVAL;
    const Shape s = shape_of(p);
    NEGF_TRY(check_sigma(sigma_r, s.n, true));
    if (!ctx->ws) return NEGF_ENOWORKSPACE;
    Workspace W = carve_workspace(ctx->ws, s.n, s.b, s.ne);
    if (W.bytes > ctx->ws_bytes) return NEGF_ENOWORKSPACE;
    ctx->sweep_valid = false;
    cplx* GRd = (cplx*)GR_diag_; cplx* GRu = (cplx*)GR_upper_; cplx* GRl = (cplx*)GR_lower_;
    const int b = s.b, ne = s.ne, n = s.n;
    cplx *T0 = W.T[0], *T1 = W.T[1], *T2 = W.T[2], *T3 = W.T[3], *T4 = W.T[4], *T5 = W.T[5];
    NEGF_TRY(ew_fill_int(ctx, info, ne, 0));

    // S3 forward: g_0 = A_00^-1 ; g_i = (A_ii - A_{i,i-1} g_{i-1} A_{i-1,i})^-1
    for (int i = 0; i < n; i++) {
        cplx* gi = W.g + s.bb * i;
        if (i == 0) {
            NEGF_TRY(assemble_a(ctx, p, sigma_r, s, 0, 0, gi, s.sn));
        } else {
            cplx* Yi = W.Y + s.bb * (i - 1);
            NEGF_TRY(assemble_a(ctx, p, sigma_r, s, 0, i, T0, s.sb));
            NEGF_TRY(assemble_a(ctx, p, sigma_r, s, 2, i - 1, T1, s.sb));      // A_{i,i-1}
            NEGF_TRY(assemble_a(ctx, p, sigma_r, s, 1, i - 1, T2, s.sb));      // A_{i-1,i}
            NEGF_TRY(zgemm_bb(ctx, 0, 0, b, ONE, T1, s.sb, W.g + s.bb * (i - 1), s.sn, ZERO, nullptr, 0,
                              Yi, s.sm, ne, nullptr));                          // Y_{i-1} = A_{i,i-1} g_{i-1}
            NEGF_TRY(zgemm_bb(ctx, 0, 0, b, MONE, Yi, s.sm, T2, s.sb, ONE, T0, s.sb, gi, s.sn, ne, nullptr));
        }
        NEGF_TRY(zinv_launch(ctx, b, gi, s.sn, ne, W.inv, info, i + 1, nullptr));
    }
    // S4 backward
    NEGF_TRY(ew_copy(ctx, s.bb, ne, GRd + s.bb * (n - 1), s.sn, W.g + s.bb * (n - 1), s.sn, nullptr));
    cplx* col = T3; cplx* coln = T5;
    if (GR_corner_) NEGF_TRY(ew_copy(ctx, s.bb, ne, col, s.sb, W.g + s.bb * (n - 1), s.sn, nullptr));
    for (int i = n - 2; i >= 0; i--) {
        cplx* gi = W.g + s.bb * i; cplx* Xi = W.X + s.bb * i; cplx* Yi = W.Y + s.bb * i;
        cplx* Gnext = GRd + s.bb * (i + 1);
        NEGF_TRY(assemble_a(ctx, p, sigma_r, s, 1, i, T2, s.sb));                              // A_{i,i+1}
        NEGF_TRY(zgemm_bb(ctx, 0, 0, b, ONE, gi, s.sn, T2, s.sb, ZERO, nullptr, 0, Xi, s.sm, ne, nullptr));
        cplx* Gu = GRu ? GRu + s.bb * i : T4; long long sGu = GRu ? s.sm : s.sb;
        NEGF_TRY(zgemm_bb(ctx, 0, 0, b, MONE, Xi, s.sm, Gnext, s.sn, ZERO, nullptr, 0, Gu, sGu, ne, nullptr));
        if (GRl) NEGF_TRY(zgemm_bb(ctx, 0, 0, b, MONE, Gnext, s.sn, Yi, s.sm, ZERO, nullptr, 0,
                                   GRl + s.bb * i, s.sm, ne, nullptr));
        NEGF_TRY(zgemm_bb(ctx, 0, 0, b, MONE, Gu, sGu, Yi, s.sm, ONE, gi, s.sn, GRd + s.bb * i, s.sn, ne, nullptr));
        if (GR_corner_) {
            NEGF_TRY(zgemm_bb(ctx, 0, 0, b, MONE, Xi, s.sm, col, s.sb, ZERO, nullptr, 0, coln, s.sb, ne, nullptr));
            cplx* t = col; col = coln; coln = t;
        }
    }
    if (GR_corner_) NEGF_TRY(ew_copy(ctx, s.bb, ne, (cplx*)GR_corner_, s.sb, col, s.sb, nullptr));
    if (flags & NEGF_KEEP_SWEEP) { ctx->sweep_valid = true; ctx->sw_n = n; ctx->sw_b = b; ctx->sw_ne = ne; }
    return NEGF_OK;
}

namespace {

// S5 + S6 for one of </>.  GXd [NE][n][b][b] required, GXu [NE][n-1][b][b] optional.
int lesser_greater_one(negf_ctx* ctx, const negf_problem* p, const negf_sigma* sr, const negf_sigma* sx,
                       const Shape& s, Workspace& W, const cplx* GRd, cplx* GXd, cplx* GXu) {
    const int b = s.b, ne = s.ne, n = s.n;
    cplx *T0 = W.T[0], *T1 = W.T[1], *T2 = W.T[2], *T3 = W.T[3], *T4 = W.T[4], *T5 = W.T[5],
         *T6 = W.T[6], *T7 = W.T[7], *T8 = W.T[8];
    bool zero_blk;
    // S5 forward: g^x_0 = g_0 B_00 g_0^H
    NEGF_TRY(assemble_b(ctx, sx, s, 0, 0, T0, &zero_blk));
    NEGF_TRY(zgemm_bb(ctx, 0, 0, b, ONE, W.g, s.sn, T0, s.sb, ZERO, nullptr, 0, T1, s.sb, ne, nullptr));
    NEGF_TRY(zgemm_bb(ctx, 0, 1, b, ONE, T1, s.sb, W.g, s.sn, ZERO, nullptr, 0, W.gx, s.sn, ne, nullptr));
    for (int i = 1; i < n; i++) {
        cplx* gi = W.g + s.bb * i; cplx* Yp = W.Y + s.bb * (i - 1);
        NEGF_TRY(assemble_b(ctx, sx, s, 0, i, T0, &zero_blk));                    // B_ii
        NEGF_TRY(assemble_a(ctx, p, sr, s, 2, i - 1, T1, s.sb));                  // A_{i,i-1}
        NEGF_TRY(zgemm_bb(ctx, 0, 0, b, ONE, T1, s.sb, W.gx + s.bb * (i - 1), s.sn, ZERO, nullptr, 0,
                          T2, s.sb, ne, nullptr));                                // A_{i,i-1} g^x_{i-1}
        NEGF_TRY(zgemm_bb(ctx, 0, 1, b, ONE, T2, s.sb, T1, s.sb, ONE, T0, s.sb, T3, s.sb, ne, nullptr));
        NEGF_TRY(assemble_b(ctx, sx, s, 1, i - 1, T4, &zero_blk));                // B_{i-1,i}
        if (!zero_blk) {
            // - Y B_up - B_low Y^H = -(W - W^H), W = Y_{i-1} B_{i-1,i}   (B_low = -B_up^H)
            NEGF_TRY(zgemm_bb(ctx, 0, 0, b, ONE, Yp, s.sm, T4, s.sb, ZERO, nullptr, 0, T5, s.sb, ne, nullptr));
            NEGF_TRY(ew_antiherm_add(ctx, b, ne, T3, s.sb, T3, s.sb, T5, s.sb, -1.0));
        }
        NEGF_TRY(zgemm_bb(ctx, 0, 0, b, ONE, gi, s.sn, T3, s.sb, ZERO, nullptr, 0, T2, s.sb, ne, nullptr));
        NEGF_TRY(zgemm_bb(ctx, 0, 1, b, ONE, T2, s.sb, gi, s.sn, ZERO, nullptr, 0, W.gx + s.bb * i, s.sn, ne, nullptr));
    }
    // S6 backward
    NEGF_TRY(ew_copy(ctx, s.bb, ne, GXd + s.bb * (n - 1), s.sn, W.gx + s.bb * (n - 1), s.sn, nullptr));
    for (int i = n - 2; i >= 0; i--) {
        cplx* gi = W.g + s.bb * i; cplx* gxi = W.gx + s.bb * i; cplx* Xi = W.X + s.bb * i;
        const cplx* GRn = GRd + s.bb * (i + 1); cplx* GXn = GXd + s.bb * (i + 1);
        NEGF_TRY(assemble_a(ctx, p, sr, s, 2, i, T1, s.sb));                      // A_{i+1,i}
        NEGF_TRY(zgemm_bb(ctx, 0, 1, b, MONE, gxi, s.sn, T1, s.sb, ZERO, nullptr, 0, T2, s.sb, ne, nullptr));
        NEGF_TRY(assemble_b(ctx, sx, s, 1, i, T4, &zero_blk));                    // B_{i,i+1}
        if (!zero_blk)
            NEGF_TRY(zgemm_bb(ctx, 0, 0, b, ONE, gi, s.sn, T4, s.sb, ONE, T2, s.sb, T2, s.sb, ne, nullptr));
        NEGF_TRY(zgemm_bb(ctx, 0, 1, b, ONE, T2, s.sb, GRn, s.sn, ZERO, nullptr, 0, T3, s.sb, ne, nullptr));  // Q
        NEGF_TRY(zgemm_bb(ctx, 0, 0, b, ONE, Xi, s.sm, GXn, s.sn, ZERO, nullptr, 0, T5, s.sb, ne, nullptr));  // R
        cplx* Gu = GXu ? GXu + s.bb * i : T6; long long sGu = GXu ? s.sm : s.sb;
        NEGF_TRY(ew_sub(ctx, b, ne, Gu, sGu, T3, s.sb, T5, s.sb));                // G^x_{i,i+1} = Q - R
        NEGF_TRY(zgemm_bb(ctx, 0, 1, b, ONE, Xi, s.sm, Gu, sGu, ZERO, nullptr, 0, T7, s.sb, ne, nullptr));    // V
        NEGF_TRY(zgemm_bb(ctx, 0, 1, b, MONE, T5, s.sb, Xi, s.sm, ONE, gxi, s.sn, T8, s.sb, ne, nullptr));    // Z
        NEGF_TRY(ew_antiherm_add(ctx, b, ne, GXd + s.bb * i, s.sn, T8, s.sb, T7, s.sb, 1.0));
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
    Workspace W = carve_workspace(ctx->ws, s.n, s.b, s.ne);
    if (W.bytes > ctx->ws_bytes) return NEGF_ENOWORKSPACE;
    if (!ctx->sweep_valid || ctx->sw_n != s.n || ctx->sw_b != s.b || ctx->sw_ne != s.ne) return NEGF_ENOSTATE;
    NEGF_TRY(ew_fill_int(ctx, info, s.ne, 0));
    if (sigma_lesser)
        NEGF_TRY(lesser_greater_one(ctx, p, sigma_r, sigma_lesser, s, W, (const cplx*)GR_diag, (cplx*)GL_diag, (cplx*)GL_upper));
    if (sigma_greater)
        NEGF_TRY(lesser_greater_one(ctx, p, sigma_r, sigma_greater, s, W, (const cplx*)GR_diag, (cplx*)GG_diag, (cplx*)GG_upper));
    return NEGF_OK;
}
