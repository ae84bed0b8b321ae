// Two-sided RGF sweeps (the P = 2 case of the paper's Fig. 2, PAPER.md:66,
// inside one GPU).  Used in the latency-bound small-block regime (b <= NEGF_PAIR_MAX_B), where the
// time of a sweep is the LENGTH of its sequential chain: blocks 0 .. m-1 are eliminated from the
// left and blocks n-1 .. m+1 from the right, concurrently on two CUDA streams, and meet in the
// middle block m = n/2 - no fill-in, same selected blocks, chains half as long.
//
//   left   gL_i = (A_ii - A_{i,i-1} gL_{i-1} A_{i-1,i})^-1,  Y_i  = A_{i+1,i} gL_i,  X_i  = gL_i A_{i,i+1}   (i < m)
//   right  gR_i = (A_ii - A_{i,i+1} gR_{i+1} A_{i+1,i})^-1,  YR_i = A_{i-1,i} gR_i,  XR_i = gR_i A_{i,i-1}   (i > m)
//   middle G_mm = (A_mm - Y_{m-1} A_{m-1,m} - YR_{m+1} A_{m+1,m})^-1
//   outwards, i = m-1 .. 0:   G_{i,i+1} = -X_i G_{i+1,i+1}, G_{i+1,i} = -G_{i+1,i+1} Y_i, G_ii = gL_i - G_{i,i+1} Y_i
//             i = m+1 .. n-1: G_{i,i-1} = -XR_i G_{i-1,i-1}, G_{i-1,i} = -G_{i-1,i-1} YR_i, G_ii = gR_i - G_{i,i-1} YR_i
//   corner    G_{0,n-1} = [(-X_0) .. (-X_{m-1})] G_mm [(-YR_{m+1}) .. (-YR_{n-1})]   (third stream)
// Storage: the g family holds gL_i (i < m), G_mm and gR_i (i > m); X_i / Y_i sit at index i of their
// families, XR_i / YR_i at index i-1 (disjoint ranges).  The lesser / greater sweeps mirror the
// hoisted one-sided forms of rgf.cu in the same way (formulas at the functions).
#include "rgf_common.cuh"

using namespace rgfc;

#define NEGF_CU(ctx, expr) NEGF_CUDA_CHECK(ctx, expr)

int rgf2_retarded(negf_ctx* ctx, const negf_problem* p, const Shape& s, const Workspace& W, const Fams& F,
                  cplx* GRd_, cplx* GRu_, cplx* GRl_, cplx* GRcorner_, int* info) {
    (void)p;
    const int n = s.n, ne = s.ne, b = s.b, m = n / 2;
    const cplx sg = real(F.sgn), nsg = real(-F.sgn);
    const Opnd GRd = {GRd_, s.sn, s.sb, 0};
    StreamFork sf(ctx);
    auto inv = [&](int i) { return zinv_launch(ctx, b, W.g + s.bb * i, s.sn, ne, W.inv_side(ctx->stream != sf.main), info, i + 1, nullptr); };

    // ---- forward: left chain on the caller's stream, right chain on side stream 0
    NEGF_CU(ctx, sf.fork(0));
    const int steps = max(m, n - 1 - m);
    for (int q = 0; q < steps; q++) {
        const int iL = q, iR = n - 1 - q;
        if (iL < m) {
            sf.use_main();
            if (iL > 0) {
                NEGF_TRY(zgemm_launch(ctx, gemm_one(s, sg, F.AL, iL - 1, F.g, iL - 1, ZERO, nullptr, 0, F.Y, iL - 1)));
                NEGF_TRY(zgemm_launch(ctx, gemm_one(s, nsg, F.Y, iL - 1, F.AU, iL - 1, ONE, &F.g, iL, F.g, iL)));
            }
            NEGF_TRY(inv(iL));
        }
        if (iR > m) {
            sf.use_side(0);
            if (iR < n - 1) {     // YR_{i+1} = A_{i,i+1} gR_{i+1} (index i) ; A_ii -= YR_{i+1} A_{i+1,i}
                NEGF_TRY(zgemm_launch(ctx, gemm_one(s, sg, F.AU, iR, F.g, iR + 1, ZERO, nullptr, 0, F.Y, iR)));
                NEGF_TRY(zgemm_launch(ctx, gemm_one(s, nsg, F.Y, iR, F.AL, iR, ONE, &F.g, iR, F.g, iR)));
            }
            NEGF_TRY(inv(iR));
        }
    }
    // couplings into the middle block, X / XR families (hoisted, batched over the block index)
    sf.use_main();
    if (m > 0) {
        NEGF_TRY(zgemm_launch(ctx, gemm_one(s, sg, F.AL, m - 1, F.g, m - 1, ZERO, nullptr, 0, F.Y, m - 1)));
        NEGF_TRY(zgemm_launch(ctx, gemm_one(s, nsg, F.Y, m - 1, F.AU, m - 1, ONE, &F.g, m, F.g, m)));
        NEGF_TRY(launch_fam(ctx, s, sg, F.g, 0, F.AU, 0, ZERO, nullptr, 0, F.X, 0, m));                      // X_i, i < m
    }
    if (m < n - 1) {
        sf.use_side(0);
        NEGF_TRY(zgemm_launch(ctx, gemm_one(s, sg, F.AU, m, F.g, m + 1, ZERO, nullptr, 0, F.Y, m)));         // YR_{m+1}
        NEGF_TRY(launch_fam(ctx, s, sg, F.g, m + 1, F.AL, m, ZERO, nullptr, 0, F.X, m, n - 1 - m));          // XR_i, i > m
        NEGF_CU(ctx, sf.join(0));
        sf.use_main();
        NEGF_TRY(zgemm_launch(ctx, gemm_one(s, nsg, F.Y, m, F.AL, m, ONE, &F.g, m, F.g, m)));
    } else {
        NEGF_CU(ctx, sf.join(0));
        sf.use_main();
    }
    // ---- corner chains on side stream 1 (they need only X / YR): PL = prod(-X_i), PR = prod(-YR_j)
    const bool corner = GRcorner_ != nullptr;
    const int nl = m, nr = n - 1 - m;                 // factors in PL / PR
    cplx *PL[2] = {W.T[7], W.T[8]}, *PR[2] = {W.T[9], W.T[10]};
    int pl = 0, pr = 0;                               // buffers holding the current products
    if (corner && n > 1) {
        NEGF_CU(ctx, sf.fork(1));
        sf.use_side(1);
        const Opnd Yf = F.Y;
        for (int k = 1; k < max(nl, nr); k++) {
            GemmGroup grp; grp.ng = 0;
            if (k < nl) {
                const Opnd Ain = (k == 1) ? Opnd{F.X.p, F.X.se, F.X.si, 0} : Opnd{PL[pl], s.sb, 0, 0};
                grp.g[grp.ng++] = gemm_one(s, k == 1 ? ONE : MONE, Ain, k == 1 ? 0 : 0, F.X, k, ZERO, nullptr, 0, Opnd{PL[pl ^ (k > 1)], s.sb, 0, 0}, 0);
                if (k > 1) pl ^= 1;
            }
            if (k < nr) {
                const Opnd Ain = (k == 1) ? Opnd{Yf.p + (size_t)m * s.bb, Yf.se, Yf.si, 0} : Opnd{PR[pr], s.sb, 0, 0};
                grp.g[grp.ng++] = gemm_one(s, k == 1 ? ONE : MONE, Ain, 0, Yf, m + k, ZERO, nullptr, 0, Opnd{PR[pr ^ (k > 1)], s.sb, 0, 0}, 0);
                if (k > 1) pr ^= 1;
            }
            if (grp.ng) NEGF_TRY(zgemm_launch_group(ctx, grp));
        }
        sf.use_main();
    }
    // ---- middle block
    NEGF_TRY(inv(m));
    NEGF_TRY(ew_copy(ctx, s.bb, ne, GRd_ + s.bb * m, s.sn, W.g + s.bb * m, s.sn, nullptr));
    if (corner && n == 1) NEGF_TRY(ew_copy(ctx, s.bb, ne, GRcorner_, s.sb, W.g, s.sn, nullptr));
    if (n == 1) return NEGF_OK;

    // ---- corner = PL G_mm PR (PL = I when m = 0, PR = I when m = n-1)
    if (corner) {
        NEGF_CU(ctx, sf.side_waits_main(1));          // G_mm (and the rest of main so far)
        sf.use_side(1);
        const Opnd Gm = {W.g + s.bb * m, s.sn, 0, 0};
        const Opnd PLo = (nl == 1) ? Opnd{F.X.p, F.X.se, 0, 0} : Opnd{PL[pl], s.sb, 0, 0};
        const Opnd PRo = (nr == 1) ? Opnd{F.Y.p + (size_t)m * s.bb, F.Y.se, 0, 0} : Opnd{PR[pr], s.sb, 0, 0};
        // sign bookkeeping: a single factor is stored without its minus sign
        const cplx sl = (nl == 1) ? MONE : ONE, sr = (nr == 1) ? MONE : ONE;
        const Opnd Tm = {W.T[11], s.sb, 0, 0}, Co = {GRcorner_, s.sb, 0, 0};
        if (nl > 0 && nr > 0) {
            NEGF_TRY(zgemm_launch(ctx, gemm_one(s, sl, PLo, 0, Gm, 0, ZERO, nullptr, 0, Tm, 0)));
            NEGF_TRY(zgemm_launch(ctx, gemm_one(s, sr, Tm, 0, PRo, 0, ZERO, nullptr, 0, Co, 0)));
        } else if (nl > 0) {
            NEGF_TRY(zgemm_launch(ctx, gemm_one(s, sl, PLo, 0, Gm, 0, ZERO, nullptr, 0, Co, 0)));
        } else {
            NEGF_TRY(zgemm_launch(ctx, gemm_one(s, sr, Gm, 0, PRo, 0, ZERO, nullptr, 0, Co, 0)));
        }
        sf.use_main();
    }

    // ---- outwards: left half on the caller's stream, right half on side stream 0
    NEGF_CU(ctx, sf.fork(0));
    const Opnd GRu = GRu_ ? Opnd{GRu_, s.sm, s.sb, 0} : Opnd{W.T[4], s.sb, 0, 0};      // left chain needs G_{i,i+1}
    const Opnd GRl = GRl_ ? Opnd{GRl_, s.sm, s.sb, 0} : Opnd{W.T[6], s.sb, 0, 0};      // right chain needs G_{i,i-1}
    for (int q = 1; q <= max(m, n - 1 - m); q++) {
        const int iL = m - q, iR = m + q;
        if (iL >= 0) {
            sf.use_main();
            GemmGroup grp; grp.ng = 0;
            grp.g[grp.ng++] = gemm_one(s, MONE, F.X, iL, GRd, iL + 1, ZERO, nullptr, 0, GRu, GRu_ ? iL : 0);
            if (GRl_) grp.g[grp.ng++] = gemm_one(s, MONE, GRd, iL + 1, F.Y, iL, ZERO, nullptr, 0, GRl, iL);
            NEGF_TRY(zgemm_launch_group(ctx, grp));
            NEGF_TRY(zgemm_launch(ctx, gemm_one(s, MONE, GRu, GRu_ ? iL : 0, F.Y, iL, ONE, &F.g, iL, GRd, iL)));
        }
        if (iR <= n - 1) {
            sf.use_side(0);
            GemmGroup grp; grp.ng = 0;
            grp.g[grp.ng++] = gemm_one(s, MONE, F.X, iR - 1, GRd, iR - 1, ZERO, nullptr, 0, GRl, GRl_ ? iR - 1 : 0);   // G_{i,i-1}
            if (GRu_) grp.g[grp.ng++] = gemm_one(s, MONE, GRd, iR - 1, F.Y, iR - 1, ZERO, nullptr, 0, GRu, iR - 1);    // G_{i-1,i}
            NEGF_TRY(zgemm_launch_group(ctx, grp));
            NEGF_TRY(zgemm_launch(ctx, gemm_one(s, MONE, GRl, GRl_ ? iR - 1 : 0, F.Y, iR - 1, ONE, &F.g, iR, GRd, iR)));
        }
    }
    sf.use_main();
    if (corner) NEGF_CU(ctx, sf.join(1));
    NEGF_CU(ctx, sf.join(0));
    return NEGF_OK;
}

namespace {

// gx_i (+)= g_i B g_i^H for a boundary block B on block i
int boundary_w(negf_ctx* ctx, const Shape& s, const Fams& F, const Workspace& W, const cplx* bnd, int i, bool accumulate) {
    const Opnd Bn = {bnd, s.sb, 0, 0}, T = {W.T[0], s.sb, 0, 0};
    NEGF_TRY(zgemm_launch(ctx, gemm_one(s, ONE, F.g, i, Bn, 0, ZERO, nullptr, 0, T, 0)));
    return zgemm_launch(ctx, gemm_one(s, ONE, T, 0, dag(F.g), i, accumulate ? ONE : ZERO, accumulate ? &F.gx : nullptr, i, F.gx, i));
}

int zero_block(negf_ctx* ctx, const Shape& s, cplx* fam, int i) {
    NEGF_CUDA_CHECK(ctx, cudaMemset2DAsync(fam + s.bb * i, (size_t)s.sn * sizeof(cplx), 0, s.bb * sizeof(cplx), s.ne, ctx->stream));
    return NEGF_OK;
}

}  // namespace

// Lesser / greater, two-sided (B = Sigma^x, anti-Hermitian; Bu[i] = B_{i,i+1}, B_{i+1,i} = -Bu[i]^H):
//   W_i    = g_i [B_ii - (V_i - V_i^H) + (V'_i - V'_i^H)] g_i^H,  V_i = Y_{i-1} Bu[i-1] (1 <= i <= m),
//            V'_i = YR_{i+1} Bu[i]^H (m <= i <= n-2), with g_m = G_mm                (all blocks, batched)
//   left   g^x_i = W_i + Z_i g^x_{i-1} Z_i^H,   Z_i  = g_i A_{i,i-1}   (i = 1 .. m-1)
//   right  g^x_i = W_i + ZR_i g^x_{i+1} ZR_i^H, ZR_i = g_i A_{i,i+1}   (i = n-2 .. m+1)
//   middle G^x_mm = W_m + Z_m g^x_{m-1} Z_m^H + ZR_m g^x_{m+1} ZR_m^H
//   outwards, left  (rgf.cu S6): G^x_{i,i+1} = Q_i - X_i G^x_{i+1,i+1},  G^x_ii = P_i + X_i (G^x_{i,i+1})^H
//   outwards, right (mirror, written for the UPPER block that is stored):
//       T2R_i = -g^x_i A_{i-1,i}^H - g_i Bu[i-1]^H,   QU_i = -G^R_{i-1,i-1} T2R_i^H,   PR_i = g^x_i + QU_i^H XR_i^H,
//       G^x_{i-1,i} = QU_i - G^x_{i-1,i-1} XR_i^H,     G^x_ii = PR_i - XR_i G^x_{i-1,i}
int rgf2_lesser_greater_one(negf_ctx* ctx, const negf_sigma* sx, const Shape& s, const Workspace& W, const Fams& F,
                            const cplx* GRd_, cplx* GXd_, cplx* GXu_) {
    const int n = s.n, ne = s.ne, b = s.b, m = n / 2;
    const cplx sg = real(F.sgn), nsg = real(-F.sgn);
    const Opnd GRd = {GRd_, s.sn, s.sb, 0}, GXd = {GXd_, s.sn, s.sb, 0};
    const Opnd Qf = GXu_ ? Opnd{GXu_, s.sm, s.sb, 0} : Opnd{W.Q, s.sn, s.sb, 0};
    const bool bt = sx->kind == NEGF_SIGMA_BT;
    const Opnd Su = {(const cplx*)sx->upper, s.sm, s.sb, 0};
    StreamFork sf(ctx);

    // ---- W family, straight into the gx family
    bool have_w = false;
    if (sx->kind == NEGF_SIGMA_SCALAR) {
        NEGF_TRY(launch_fam(ctx, s, ONE, F.g, 0, dag(F.g), 0, ZERO, nullptr, 0, F.gx, 0, n, (const cplx*)sx->scalar));
        have_w = true;
    } else if (bt) {
        NEGF_TRY(ew_copy(ctx, s.bb * n, ne, W.gx, s.sn, (const cplx*)sx->diag, s.sn, nullptr));
        if (n > 1) {
            if (m >= 1) NEGF_TRY(launch_fam(ctx, s, ONE, F.Y, 0, Su, 0, ZERO, nullptr, 0, F.Q, 1, m));                   // V_i -> Q[i]
            if (m <= n - 2) NEGF_TRY(launch_fam(ctx, s, ONE, F.Y, m, dag(Su), m, ZERO, nullptr, 0, F.Z, m, n - 1 - m)); // V'_i -> Z[i]
            for (int i = 1; i <= m; i++)
                NEGF_TRY(ew_antiherm_add(ctx, b, ne, W.gx + s.bb * i, s.sn, W.gx + s.bb * i, s.sn, W.Q + s.bb * i, s.sn, -1.0));
            for (int i = m; i <= n - 2; i++)
                NEGF_TRY(ew_antiherm_add(ctx, b, ne, W.gx + s.bb * i, s.sn, W.gx + s.bb * i, s.sn, W.Z + s.bb * i, s.sm, 1.0));
        }
        NEGF_TRY(launch_fam(ctx, s, ONE, F.g, 0, F.gx, 0, ZERO, nullptr, 0, F.Q, 0, n));
        NEGF_TRY(launch_fam(ctx, s, ONE, F.Q, 0, dag(F.g), 0, ZERO, nullptr, 0, F.gx, 0, n));
        have_w = true;
    }
    bool w_first = have_w, w_last = have_w;             // W present on block 0 / n-1
    if (sx->left) { NEGF_TRY(boundary_w(ctx, s, F, W, (const cplx*)sx->left, 0, w_first)); w_first = true; if (n == 1) w_last = true; }
    if (sx->right) { NEGF_TRY(boundary_w(ctx, s, F, W, (const cplx*)sx->right, n - 1, w_last)); w_last = true; if (n == 1) w_first = true; }
    auto has_w = [&](int i) { return i == 0 ? w_first : (i == n - 1 ? w_last : have_w); };

    // ---- Z_i (i = 1 .. m, index i-1) and ZR_i (i = m .. n-2, index i)
    if (m >= 1) NEGF_TRY(launch_fam(ctx, s, sg, F.g, 1, F.AL, 0, ZERO, nullptr, 0, F.Z, 0, m));
    if (m <= n - 2) NEGF_TRY(launch_fam(ctx, s, sg, F.g, m, F.AU, m, ZERO, nullptr, 0, F.Z, m, n - 1 - m));
    if (m >= 1 && !has_w(0)) NEGF_TRY(zero_block(ctx, s, W.gx, 0));
    if (n - 1 > m && !has_w(n - 1)) NEGF_TRY(zero_block(ctx, s, W.gx, n - 1));

    // ---- the two connected chains, concurrently
    NEGF_CU(ctx, sf.fork(0));
    const Opnd TL = {W.T[1], s.sb, 0, 0}, TR = {W.T[2], s.sb, 0, 0};
    for (int q = 1; q < max(m, n - 1 - m); q++) {
        const int iL = q, iR = n - 1 - q;
        if (iL < m) {
            sf.use_main();
            const bool w = has_w(iL);
            NEGF_TRY(zgemm_launch(ctx, gemm_one(s, ONE, F.Z, iL - 1, F.gx, iL - 1, ZERO, nullptr, 0, TL, 0)));
            NEGF_TRY(zgemm_launch(ctx, gemm_one(s, ONE, TL, 0, dag(F.Z), iL - 1, w ? ONE : ZERO, w ? &F.gx : nullptr, iL, F.gx, iL)));
        }
        if (iR > m) {
            sf.use_side(0);
            const bool w = has_w(iR);
            NEGF_TRY(zgemm_launch(ctx, gemm_one(s, ONE, F.Z, iR, F.gx, iR + 1, ZERO, nullptr, 0, TR, 0)));
            NEGF_TRY(zgemm_launch(ctx, gemm_one(s, ONE, TR, 0, dag(F.Z), iR, w ? ONE : ZERO, w ? &F.gx : nullptr, iR, F.gx, iR)));
        }
    }
    NEGF_CU(ctx, sf.join(0));
    sf.use_main();
    // ---- middle block
    {
        bool acc = has_w(m);
        if (m >= 1) {
            NEGF_TRY(zgemm_launch(ctx, gemm_one(s, ONE, F.Z, m - 1, F.gx, m - 1, ZERO, nullptr, 0, TL, 0)));
            NEGF_TRY(zgemm_launch(ctx, gemm_one(s, ONE, TL, 0, dag(F.Z), m - 1, acc ? ONE : ZERO, acc ? &F.gx : nullptr, m, F.gx, m)));
            acc = true;
        }
        if (m <= n - 2) {
            NEGF_TRY(zgemm_launch(ctx, gemm_one(s, ONE, F.Z, m, F.gx, m + 1, ZERO, nullptr, 0, TR, 0)));
            NEGF_TRY(zgemm_launch(ctx, gemm_one(s, ONE, TR, 0, dag(F.Z), m, acc ? ONE : ZERO, acc ? &F.gx : nullptr, m, F.gx, m)));
            acc = true;
        }
        if (!acc) NEGF_TRY(zero_block(ctx, s, W.gx, m));
    }
    NEGF_TRY(ew_copy(ctx, s.bb, ne, GXd_ + s.bb * m, s.sn, W.gx + s.bb * m, s.sn, nullptr));
    if (n == 1) return NEGF_OK;

    // ---- outwards: hoisted products and chains, left half on the caller's stream, right half on side 0
    NEGF_CU(ctx, sf.fork(0));
    if (m >= 1) {
        sf.use_main();
        NEGF_TRY(launch_fam(ctx, s, nsg, F.gx, 0, dag(F.AL), 0, ZERO, nullptr, 0, F.Z, 0, m));              // T2_i
        if (bt) NEGF_TRY(launch_fam(ctx, s, ONE, F.g, 0, Su, 0, ONE, &F.Z, 0, F.Z, 0, m));
        NEGF_TRY(launch_fam(ctx, s, ONE, F.Z, 0, dag(GRd), 1, ZERO, nullptr, 0, Qf, 0, m));                  // Q_i
        NEGF_TRY(launch_fam(ctx, s, MONE, Qf, 0, dag(F.X), 0, ONE, &F.gx, 0, GXd, 0, m));                    // P_i
    }
    if (m <= n - 2) {
        const int cnt = n - 1 - m;
        sf.use_side(0);
        NEGF_TRY(launch_fam(ctx, s, nsg, F.gx, m + 1, dag(F.AU), m, ZERO, nullptr, 0, F.Z, m, cnt));         // T2R_i
        if (bt) NEGF_TRY(launch_fam(ctx, s, MONE, F.g, m + 1, dag(Su), m, ONE, &F.Z, m, F.Z, m, cnt));
        NEGF_TRY(launch_fam(ctx, s, MONE, GRd, m, dag(F.Z), m, ZERO, nullptr, 0, Qf, m, cnt));               // QU_i
        NEGF_TRY(launch_fam(ctx, s, ONE, dag(Qf), m, dag(F.X), m, ONE, &F.gx, m + 1, GXd, m + 1, cnt));      // PR_i
    }
    for (int q = 1; q <= max(m, n - 1 - m); q++) {
        const int iL = m - q, iR = m + q;
        if (iL >= 0) {
            sf.use_main();
            NEGF_TRY(zgemm_launch(ctx, gemm_one(s, MONE, F.X, iL, GXd, iL + 1, ONE, &Qf, iL, Qf, iL)));      // G^x_{i,i+1}
            NEGF_TRY(zgemm_launch(ctx, gemm_one(s, ONE, F.X, iL, dag(Qf), iL, ONE, &GXd, iL, GXd, iL)));     // G^x_ii
        }
        if (iR <= n - 1) {
            sf.use_side(0);
            NEGF_TRY(zgemm_launch(ctx, gemm_one(s, MONE, GXd, iR - 1, dag(F.X), iR - 1, ONE, &Qf, iR - 1, Qf, iR - 1)));   // G^x_{i-1,i}
            NEGF_TRY(zgemm_launch(ctx, gemm_one(s, MONE, F.X, iR - 1, Qf, iR - 1, ONE, &GXd, iR, GXd, iR)));              // G^x_ii
        }
    }
    sf.use_main();
    NEGF_CU(ctx, sf.join(0));
    return NEGF_OK;
}
