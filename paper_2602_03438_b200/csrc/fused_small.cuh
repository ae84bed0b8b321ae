// Resident small-block regime (fused_small.cu): argument blocks of the three chain kernels.
#pragma once
#include "common.cuh"

constexpr int NEGF_FUSED_MAX_B = 32;      // whole chain of one energy in one CTA up to this block size
// The resident kernels run one CTA per energy, each walking its chain alone.  Up to b = 16 they win at every batch size
// (two CTAs per SM; n = 32, 1184 energies: 6.4 ms against 8.9 ms for the batched lock-step launches, measured with one
// CTA per SM); for 16 < b <= 32 (one CTA per SM, FP64-pipe-bound products) only while the batch fits one wave of CTAs
// (148 energies: 2.9 against 3.1 ms; 296: 5.7 against 5.0 ms).  NEGF_OPT_FUSED_SMALL: 0 never, 1 automatic, 2 always for b <= 32.
inline bool fused_small_regime(const negf_ctx* ctx, int b, int ne) {
    if (b > NEGF_FUSED_MAX_B || ctx->fused_small == 0) return false;
    return ctx->fused_small >= 2 || b <= 16 || ne <= ctx->num_sms;
}

// device + energy batch + retarded self-energy (what the blocks of A = z S - H - Sigma^R are assembled from)
struct FusedProblem {
    int n, b, ne;
    const cplx *Hd, *Hu, *Sd, *Su;        // as negf_problem (Sd / Su NULL: S = I)
    const double* energy; double eta;
    const int* kidx;                      // k-point index per batch entry or NULL
    int sr_kind;                          // NEGF_SIGMA_* of Sigma^R_S
    const cplx *sr_scalar, *sr_diag, *sr_upper, *sr_lower, *sr_left, *sr_right;
};
struct FusedRetOut {
    cplx *g, *X, *Y;                      // workspace families (one-sided layout of rgf.cu)
    cplx *GR_diag, *GR_upper, *GR_lower, *GR_corner;
    int* info;
};
struct FusedLgOne {                       // one of < / >
    int kind; const cplx *scalar, *diag, *upper, *left, *right;
    cplx *gx;                             // workspace family [ne][n][b][b] for g^x_i
    cplx *GX_diag, *GX_upper;
};
struct FusedLgArgs {
    const cplx *g, *X, *Y, *GR_diag;
    int nx; FusedLgOne x[2];
};
struct FusedLead {
    const cplx *Hd, *Hu, *Sd, *Su; long long kd, ku; int side; double mu;
    cplx *sigma_r, *gamma, *sigma_lesser, *sigma_greater, *g_surface; double* fermi; int *iters, *status;
};
struct FusedObcArgs {
    int b, ne, ns; const double* energy; double eta; const int* kidx;
    double kT, tol; int max_iter;
    FusedLead lead[2];
};
int fused_prepare(negf_ctx* ctx);
int fused_obc_launch(negf_ctx* ctx, const FusedObcArgs& a);
int fused_ret_launch(negf_ctx* ctx, const FusedProblem& P, const FusedRetOut& o);
int fused_lg_launch(negf_ctx* ctx, const FusedProblem& P, const FusedLgArgs& a);
