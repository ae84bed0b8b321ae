// Helpers shared by the one-sided (rgf.cu) and two-sided (rgf2.cu) RGF sweeps: shapes, argument
// checks, operand views of block families and GEMM argument builders.
#pragma once
#include "common.cuh"
#include "kernels.cuh"
#include "workspace.cuh"

namespace rgfc {

struct Shape { int n, b, ne; size_t bb; long long sb, sn, sm; };   // sn = n*bb, sm = (n-1)*bb

inline Shape shape_of(const negf_problem* p) {
    Shape s;
    s.n = p->n_blocks; s.b = p->block_size; s.ne = p->n_energy;
    s.bb = (size_t)s.b * s.b; s.sb = (long long)s.bb; s.sn = (long long)s.bb * s.n;
    s.sm = (long long)s.bb * (s.n - 1);
    return s;
}

inline int check_problem(const negf_ctx* ctx, const negf_problem* p) {
    if (!ctx || !p) return NEGF_EINVAL;
    if (p->n_blocks < 1 || p->block_size < 1 || p->n_energy < 1) return NEGF_EINVAL;
    if (!p->H_diag || !p->energy) return NEGF_EINVAL;
    if (p->n_blocks > 1 && !p->H_upper) return NEGF_EINVAL;
    if (p->n_blocks > 1 && ((p->S_diag == nullptr) != (p->S_upper == nullptr))) return NEGF_EINVAL;
    if (p->n_energy > 65535) return NEGF_EUNSUPPORTED;
    if (p->n_k > 1 && !p->k_index) return NEGF_EINVAL;
    return NEGF_OK;
}

// k-point batching (include/negf.h): device index per batch entry, or NULL for a single device
inline const int* kidx_of(const negf_problem* p) { return p->n_k > 1 ? p->k_index : nullptr; }

inline int check_sigma(const negf_sigma* s, int n, bool retarded) {
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

// the off-diagonal blocks of A are materialised per batch entry when they depend on it: S != I, a dense
// Sigma^R_S, or k-point batching (H_{i,i+1} differs between the entries)
inline bool needs_assembly(const negf_problem* p, const negf_sigma* sr) {
    return p->S_diag != nullptr || (sr && sr->kind == NEGF_SIGMA_BT) || p->n_k > 1;
}

// A family of blocks as a GEMM operand: block i of energy e at p + e*se + i*si, read as op(.)
struct Opnd { const cplx* p; long long se, si; int op; };
inline Opnd dag(Opnd o) { o.op ^= 1; return o; }

static const cplx ONE = {1.0, 0.0}, MONE = {-1.0, 0.0}, ZERO = {0.0, 0.0};
inline cplx real(double x) { return cmake(x, 0.0); }

// C(ic + j) = alpha op(A(ia + j)) op(B(ib + j)) + beta D(id + j), j < cnt, for all energies
inline GemmArgs gemm_fam(const Shape& s, cplx alpha, Opnd A, int ia, Opnd B, int ib, cplx beta, const Opnd* D, int id,
                  Opnd C, int ic, int cnt) {
    GemmArgs g = zgemm_bb_args(A.op, B.op, s.b, alpha, A.p + (size_t)ia * A.si, A.se, B.p + (size_t)ib * B.si, B.se, beta,
                               D ? D->p + (size_t)id * D->si : nullptr, D ? D->se : 0,
                               const_cast<cplx*>(C.p) + (size_t)ic * C.si, C.se, s.ne, nullptr);
    g.batch2 = cnt; g.sA2 = A.si; g.sB2 = B.si; g.sD2 = D ? D->si : 0; g.sC2 = C.si;
    return g;
}
inline GemmArgs gemm_one(const Shape& s, cplx alpha, Opnd A, int ia, Opnd B, int ib, cplx beta, const Opnd* D, int id,
                         Opnd C, int ic) {
    return gemm_fam(s, alpha, A, ia, B, ib, beta, D, id, C, ic, 1);
}
// families batched over (energy x i) can exceed the grid.y limit: split along i
inline int launch_fam(negf_ctx* ctx, const Shape& s, cplx alpha, Opnd A, int ia, Opnd B, int ib, cplx beta, const Opnd* D,
               int id, Opnd C, int ic, int cnt, const cplx* alpha_vec = nullptr) {
    const int chunk = max(1, 65535 / s.ne);
    for (int j = 0; j < cnt; j += chunk) {
        GemmArgs g = gemm_fam(s, alpha, A, ia + j, B, ib + j, beta, D, id + j, C, ic + j, min(chunk, cnt - j));
        g.alpha_vec = alpha_vec;
        NEGF_TRY(zgemm_launch(ctx, g));
    }
    return NEGF_OK;
}

struct Fams {                // operand views of the workspace families and of A's off-diagonal blocks
    Opnd g, X, Y, gx, Z, Q, AU, AL;
    double sgn;              // AU / AL hold sgn * A_{i,i+1} / A_{i+1,i}
};
inline Fams make_fams(const negf_problem* p, const Shape& s, const Workspace& W, bool assembled) {
    Fams f;
    f.g = {W.g, s.sn, s.sb, 0}; f.gx = {W.gx, s.sn, s.sb, 0}; f.Q = {W.Q, s.sn, s.sb, 0};
    f.X = {W.X, s.sm, s.sb, 0}; f.Y = {W.Y, s.sm, s.sb, 0}; f.Z = {W.Z, s.sm, s.sb, 0};
    if (assembled) {
        f.AU = {W.Aup, s.sm, s.sb, 0}; f.AL = {W.Alow, s.sm, s.sb, 0}; f.sgn = 1.0;
    } else {                 // A_{i,i+1} = -H_{i,i+1}, A_{i+1,i} = -H_{i,i+1}^H for every energy
        f.AU = {(const cplx*)p->H_upper, 0, s.sb, 0}; f.AL = {(const cplx*)p->H_upper, 0, s.sb, 1}; f.sgn = -1.0;
    }
    return f;
}


}  // namespace rgfc

// rgf.cu
int rgf_assemble(negf_ctx* ctx, const negf_problem* p, const negf_sigma* sigma_r, const rgfc::Shape& s,
                 const Workspace& W, bool assembled);
// rgf2.cu: two-sided sweeps, used for b <= NEGF_PAIR_MAX_B
int rgf2_retarded(negf_ctx* ctx, const negf_problem* p, const rgfc::Shape& s, const Workspace& W, const rgfc::Fams& F,
                  cplx* GRd, cplx* GRu, cplx* GRl, cplx* GRcorner, int* info);
int rgf2_lesser_greater_one(negf_ctx* ctx, const negf_sigma* sx, const rgfc::Shape& s, const Workspace& W,
                            const rgfc::Fams& F, const cplx* GRd, cplx* GXd, cplx* GXu);
