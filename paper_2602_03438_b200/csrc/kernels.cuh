// Internal declarations of the O(b^2) kernels (elementwise.cu) and observables (observables.cu).
#pragma once
#include "common.cuh"

// out[e](r,c) = [use_z ? z_e * S(r,c) : 0] - H(r,c) + coef * (blk0 + blk1 + blk2)[e](r,c)
//               + coef * scalar[e] * delta_rc,
// with X(r,c) = dagger ? conj(X[c][r]) : X[r][c] for X in {S, H} (shared by all energies),
// S == NULL && s_identity => S = I;  S == NULL && !s_identity => S = 0;  H == NULL => no H term.
struct CombineArgs {
    int b;
    const cplx* H; const cplx* S; int s_identity; int dagger; int use_z;
    const double* energy; double eta;
    const cplx* blk[3]; long long sblk[3];
    const cplx* scalar;
    double coef;
    cplx* out; long long sout;
    const int* skip;
    // family mode (nfam > 1): blockIdx.z = block index i; H, S, out and blk[t] advance by the strides
    // below per i; blk[t] contributes only to block only[t] when only[t] >= 0 (boundary blocks).
    int nfam;
    long long fH, fS, fout, fblk[3];
    int only[3];
    // k-point batching: entry e reads H + kidx[e] * kH and S + kidx[e] * kS (kidx NULL: one device)
    const int* kidx;
    long long kH, kS;
};
int ew_combine(negf_ctx* ctx, const CombineArgs& a, int batch);
// C = Z + sign * (V - V^H)   (Z may be NULL)
int ew_antiherm_add(negf_ctx* ctx, int b, int batch, cplx* C, long long sC, const cplx* Z, long long sZ,
                    const cplx* V, long long sV, double sign);
int ew_sub(negf_ctx* ctx, int b, int batch, cplx* C, long long sC, const cplx* A, long long sA,
           const cplx* B, long long sB);
int ew_copy(negf_ctx* ctx, size_t n_elems_per, int batch, cplx* dst, long long sd, const cplx* src,
            long long ss, const int* skip);
int ew_fill_int(negf_ctx* ctx, int* p, int n, int v);
int ew_max_int(negf_ctx* ctx, int* dst, const int* src, int n);   // dst = dst ? dst : src
int ew_sr_update(negf_ctx* ctx, int b, int batch, cplx* a_s, cplx* a_b, cplx* g, const cplx* lgu,
                 const cplx* ugl, const int* skip);
int ew_sr_step(negf_ctx* ctx, int b, int batch, cplx* a_s, cplx* a_b, cplx* g, const cplx* lgu, const cplx* ugl,
               const cplx* un, const cplx* ln, const double* ref, double tol, int* done, int* iters, int it,
               double* acc /*[batch][8][2]*/, unsigned* ticket /*[batch], zero*/, const int* it_dev = nullptr);
int ew_sr_cond(negf_ctx* ctx, cudaGraphConditionalHandle h, int nb, const int* done, int* it_dev, int max_iter, int step);
int ew_sr_norm(negf_ctx* ctx, int b, int batch, const cplx* u, const cplx* l, double* ref, double tol,
               int* done, int* iters, int it, int mode);
int ew_obc_finalize(negf_ctx* ctx, int b, int batch, const cplx* sigma, const double* energy, double mu,
                    double kT, cplx* gamma, cplx* sl, cplx* sg, double* fermi);
int ew_obc_status(negf_ctx* ctx, int ne, const int* done, const int* sing, const int* it_in, int* status, int* iters);
