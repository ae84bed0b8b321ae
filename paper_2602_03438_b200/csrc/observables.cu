// S7 (readings R11-R13): density, LDOS, transmission, bond and contact currents
// from the selected blocks.  O(n b^2) reductions plus two b^3 products
// for T(E).  Deterministic: no atomics, fixed reduction order.
#include "common.cuh"
#include "kernels.cuh"
#include "workspace.cuh"
#include "fused_small.cuh"

namespace {

__device__ __forceinline__ double block_sum(double v) {
    __shared__ double sh[32];
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
    __syncthreads();
    double t = 0.0;
    if (threadIdx.x < 32) {
        t = threadIdx.x < (blockDim.x >> 5) ? sh[threadIdx.x] : 0.0;
        for (int o = 16; o > 0; o >>= 1) t += __shfl_down_sync(0xffffffffu, t, o);
    }
    return t;   // valid in thread 0
}

// LDOS_i(E) = -(1/pi) Im Tr[(G^R S)_ii];  grid (n, NE)
__device__ __forceinline__ void ldos_body(int i, int e, int n, int b, const cplx* GRd, const cplx* GRu, const cplx* GRl,
                                          const cplx* Sd, const cplx* Su, const int* kidx, double* ldos) {
    const size_t bb = (size_t)b * b;
    if (kidx && Sd) { Sd += (size_t)kidx[e] * n * bb; Su += (size_t)kidx[e] * (n - 1) * bb; }   // k-point batching
    const cplx* G = GRd + ((size_t)e * n + i) * bb;
    double acc = 0.0;   // imaginary part of the trace
    if (!Sd) {
        for (int r = threadIdx.x; r < b; r += blockDim.x) acc += G[(size_t)r * b + r].y;
    } else {
        const cplx* S = Sd + (size_t)i * bb;
        for (int idx = threadIdx.x; idx < (int)bb; idx += blockDim.x) {
            int r = idx / b, c = idx % b;
            // G[r][c] * S[c][r], S Hermitian-stored as given: read S[c][r] directly
            cplx g = G[idx], s = S[(size_t)c * b + r];
            acc += g.x * s.y + g.y * s.x;
            if (i + 1 < n) {   // G_{i,i+1}[r][c] * S_{i+1,i}[c][r], S_{i+1,i} = S_up[i]^H
                cplx gu = GRu[((size_t)e * (n - 1) + i) * bb + idx], su = Su[(size_t)i * bb + idx];
                acc += -gu.x * su.y + gu.y * su.x;
            }
            if (i > 0) {       // G_{i,i-1}[r][c] * S_{i-1,i}[c][r]
                cplx gl = GRl[((size_t)e * (n - 1) + i - 1) * bb + idx], su = Su[(size_t)(i - 1) * bb + (size_t)c * b + r];
                acc += gl.x * su.y + gl.y * su.x;
            }
        }
    }
    double t = block_sum(acc);
    if (threadIdx.x == 0) ldos[(size_t)e * n + i] = -t / 3.14159265358979323846;
}
__global__ void ldos_kernel(int n, int b, const cplx* GRd, const cplx* GRu, const cplx* GRl,
                            const cplx* Sd, const cplx* Su, const int* kidx, double* ldos) {
    ldos_body(blockIdx.x, blockIdx.y, n, b, GRd, GRu, GRl, Sd, Su, kidx, ldos);
}

// density_k = sum_E w_E Im[(G^< S)_kk] / (2 pi); one warp per k; terms with row-contiguous reads.
// COLS: the third term (density_cols_kernel below) is folded into the same pass (resident small-block regime)
template <bool COLS>
__device__ __forceinline__ void density_rows_body(int warp, int n, int b, int ne, const cplx* GLd, const cplx* GLu, const cplx* Sd0,
                                                  const cplx* Su0, const int* kidx, const double* w, double* density) {
    const int lane = threadIdx.x & 31;
    if (warp >= n * b) return;
    const int i = warp / b, r = warp % b;
    const size_t bb = (size_t)b * b;
    double acc = 0.0;
    if (!Sd0) {
        // S = I: one element per energy; the lanes take the energies (a serial walk by one lane was 0.6 us per energy)
        for (int e = lane; e < ne; e += 32) acc += w[e] * GLd[((size_t)e * n + i) * bb + (size_t)r * b + r].y;
    } else
    for (int e = 0; e < ne; e++) {
        double im = 0.0;
        const cplx* G = GLd + ((size_t)e * n + i) * bb + (size_t)r * b;
        const cplx* Sd = Sd0; const cplx* Su = Su0;
        if (kidx) { Sd += (size_t)kidx[e] * n * bb; Su += (size_t)kidx[e] * (n - 1) * bb; }
        {
            const cplx* S = Sd + (size_t)i * bb + (size_t)r * b;    // S_ii[c][r] = conj(S_ii[r][c])
            for (int c = lane; c < b; c += 32) { cplx g = G[c], s = S[c]; im += -g.x * s.y + g.y * s.x; }
            if (i + 1 < n) {   // G^<_{i,i+1}[r][c] * conj(S_up[i][r][c])
                const cplx* Gu = GLu + ((size_t)e * (n - 1) + i) * bb + (size_t)r * b;
                const cplx* S2 = Su + (size_t)i * bb + (size_t)r * b;
                for (int c = lane; c < b; c += 32) { cplx g = Gu[c], s = S2[c]; im += -g.x * s.y + g.y * s.x; }
            }
            if (COLS && i > 0) {   // G^<_{i,i-1}[r][c] S_{i-1,i}[c][r], G^<_{i,i-1}[r][c] = -conj(GLu[i-1][c][r])
                const cplx* Gl = GLu + ((size_t)e * (n - 1) + i - 1) * bb;
                const cplx* S3 = Su + (size_t)(i - 1) * bb;
                for (int c = lane; c < b; c += 32) { cplx g = Gl[(size_t)c * b + r], s = S3[(size_t)c * b + r]; im += -g.x * s.y + g.y * s.x; }
            }
        }
        acc += w[e] * im;
    }
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
    if (lane == 0) density[warp] = acc / (2.0 * 3.14159265358979323846);
}
__global__ void density_rows_kernel(int n, int b, int ne, const cplx* GLd, const cplx* GLu, const cplx* Sd0,
                                    const cplx* Su0, const int* kidx, const double* w, double* density) {
    density_rows_body<false>((blockIdx.x * blockDim.x + threadIdx.x) >> 5, n, b, ne, GLd, GLu, Sd0, Su0, kidx, w, density);
}
// third term (S != I, i > 0): sum_c G^<_{i,i-1}[r][c] S_{i-1,i}[c][r], G^<_{i,i-1}[r][c] = -conj(GLu[i-1][c][r]).
// A CTA takes 32 consecutive (i, r) (threadIdx.x: coalesced down the columns) and splits the c loop over 8 slices
// (threadIdx.y), added in a fixed order at the end.  (One thread per (i, r) walking all N_E x b elements alone was
// latency-bound: 10.6 ms per 128-energy batch of configs[2] for 8.4 GB, 0.8 TB/s.)
constexpr int DC_ROWS = 32, DC_SLICES = 8;
__global__ void __launch_bounds__(DC_ROWS * DC_SLICES) density_cols_kernel(int n, int b, int ne, const cplx* GLu, const cplx* Su,
                                                                           const int* kidx, const double* w, double* density) {
    __shared__ double part[DC_SLICES][DC_ROWS + 1];
    const int k = blockIdx.x * DC_ROWS + threadIdx.x, ys = threadIdx.y;
    const bool live = k < n * b && k >= b;          // block row i = k / b > 0
    double acc = 0.0;
    if (live) {
        const int i = k / b, r = k % b;
        const size_t bb = (size_t)b * b;
        for (int e = 0; e < ne; e++) {
            const cplx* S = Su + (size_t)(i - 1) * bb + (kidx ? (size_t)kidx[e] * (n - 1) * bb : 0) + r;
            const cplx* G = GLu + ((size_t)e * (n - 1) + i - 1) * bb + r;
            double im = 0.0;
#pragma unroll 4
            for (int c = ys; c < b; c += DC_SLICES) {
                const cplx g = G[(size_t)c * b], s = S[(size_t)c * b];
                // (-conj(g)) * s = -(g.x s.x + g.y s.y) + i (-(g.x s.y) + g.y s.x)
                im += -g.x * s.y + g.y * s.x;
            }
            acc += w[e] * im;
        }
    }
    part[ys][threadIdx.x] = acc;
    __syncthreads();
    if (ys == 0 && live) {
        double t = 0.0;
#pragma unroll
        for (int q = 0; q < DC_SLICES; q++) t += part[q][threadIdx.x];
        density[k] += t / (2.0 * 3.14159265358979323846);
    }
}

// out[e] = scale * Re sum_{r,c} A[e][r][c] * conj(B[e][r][c]); grid (items, NE)
__global__ void dot_conj_kernel(int b, const cplx* A, long long sA, const cplx* B, long long sB, double scale,
                                double* out, int out_stride, int items_stride_a, int items_stride_b) {
    const int it = blockIdx.x, e = blockIdx.y;
    const cplx* a = A + (size_t)e * sA + (size_t)it * items_stride_a;
    const cplx* bp = B + (size_t)e * sB + (size_t)it * items_stride_b;
    double acc = 0.0;
    for (int idx = threadIdx.x; idx < b * b; idx += blockDim.x) { cplx x = a[idx], y = bp[idx]; acc += x.x * y.x + x.y * y.y; }
    double t = block_sum(acc);
    if (threadIdx.x == 0) out[(size_t)e * out_stride + it] = scale * t;
}

// J_i(E) = 2 Re Tr[(H_up[i] - E S_up[i]) G^<_{i+1,i}] = -2 Re sum (H - E S)[r][c] conj(GLu[r][c]); grid (n-1, NE)
__device__ __forceinline__ void bond_current_body(int i, int e, int n, int b, const cplx* Hu, const cplx* Su, const int* kidx,
                                                  const double* energy, const cplx* GLu, double* out) {
    const size_t bb = (size_t)b * b;
    const double E = energy[e];
    const size_t koff = kidx ? (size_t)kidx[e] * (n - 1) * bb : 0;
    const cplx* H = Hu + (size_t)i * bb + koff;
    const cplx* S = Su ? Su + (size_t)i * bb + koff : nullptr;
    const cplx* G = GLu + ((size_t)e * (n - 1) + i) * bb;
    double acc = 0.0;
    for (int idx = threadIdx.x; idx < (int)bb; idx += blockDim.x) {
        cplx h = H[idx];
        if (S) { cplx s = S[idx]; h.x -= E * s.x; h.y -= E * s.y; }
        cplx g = G[idx];
        acc += h.x * g.x + h.y * g.y;
    }
    double t = block_sum(acc);
    if (threadIdx.x == 0) out[(size_t)e * (n - 1) + i] = -2.0 * t;
}
__global__ void bond_current_kernel(int n, int b, const cplx* Hu, const cplx* Su, const int* kidx, const double* energy,
                                    const cplx* GLu, double* out) {
    bond_current_body(blockIdx.x, blockIdx.y, n, b, Hu, Su, kidx, energy, GLu, out);
}

// I_c(E) = Re Tr[Sigma^<_c G^>_cc - Sigma^>_c G^<_cc]; grid (2, NE)
__device__ __forceinline__ void contact_current_body(int c, int e, int n, int b, const cplx* sLl, const cplx* sLg, const cplx* sRl,
                                                     const cplx* sRg, const cplx* GLd, const cplx* GGd, double* out) {
    const size_t bb = (size_t)b * b;
    const cplx* sl = (c == 0 ? sLl : sRl) + (size_t)e * bb;
    const cplx* sg = (c == 0 ? sLg : sRg) + (size_t)e * bb;
    const int blk = c == 0 ? 0 : n - 1;
    const cplx* gl = GLd + ((size_t)e * n + blk) * bb;
    const cplx* gg = GGd + ((size_t)e * n + blk) * bb;
    double acc = 0.0;
    for (int idx = threadIdx.x; idx < (int)bb; idx += blockDim.x) {
        int r = idx / b, k = idx % b;
        cplx a = sl[idx], x = gg[(size_t)k * b + r];
        cplx d = sg[idx], y = gl[(size_t)k * b + r];
        acc += (a.x * x.x - a.y * x.y) - (d.x * y.x - d.y * y.y);
    }
    double t = block_sum(acc);
    if (threadIdx.x == 0) out[(size_t)e * 2 + c] = t;
}
__global__ void contact_current_kernel(int n, int b, const cplx* sLl, const cplx* sLg, const cplx* sRl,
                                       const cplx* sRg, const cplx* GLd, const cplx* GGd, double* out) {
    contact_current_body(blockIdx.x, blockIdx.y, n, b, sLl, sLg, sRl, sRg, GLd, GGd, out);
}

// ---- resident small-block regime (b <= 32): all of S7 in ONE launch ------------------------------------------------------
// At these sizes every observable is a fraction of a microsecond of arithmetic and the seven separate launches above
// are 48 us of launch latency (configs[0]).  One grid whose blocks take roles: LDOS (n x N_E blocks), density rows (8
// rows per block, all three terms), T(E) (one block per energy: Gamma_L G in shared memory, then the trace of
// (Gamma_L G Gamma_R) with conj(G) element by element), bond currents, contact currents.  Same formulas.
struct ObsSmallArgs {
    int n, b, ne;
    const cplx *GRd, *GRu, *GRl, *GRc, *GLd, *GLu, *GGd, *gamL, *gamR, *sLl, *sLg, *sRl, *sRg;
    const cplx *Hu, *Sd, *Su; const int* kidx; const double *energy, *w;
    double *density, *ldos, *trans, *bond, *contact;
    int n_ldos, n_dens, n_trans, n_bond, n_contact;         // blocks per role
};
__global__ void __launch_bounds__(256) obs_small_kernel(const ObsSmallArgs a) {
    __shared__ cplx tmp[32 * 33];
    int r = blockIdx.x;
    const int n = a.n, b = a.b, ne = a.ne;
    if (r < a.n_ldos) { ldos_body(r % n, r / n, n, b, a.GRd, a.GRu, a.GRl, a.Sd, a.Su, a.kidx, a.ldos); return; }
    r -= a.n_ldos;
    if (r < a.n_dens) { density_rows_body<true>(r * 8 + (threadIdx.x >> 5), n, b, ne, a.GLd, a.GLu, a.Sd, a.Su, a.kidx, a.w, a.density); return; }
    r -= a.n_dens;
    if (r < a.n_trans) {
        // T = Re Tr[Gamma_L G Gamma_R G^H] = Re sum_{rc} (Gamma_L G Gamma_R)[r][c] conj(G[r][c]),  G = G^R_{0,n-1}
        const size_t bb = (size_t)b * b;
        const cplx* gl = a.gamL + (size_t)r * bb; const cplx* gr = a.gamR + (size_t)r * bb; const cplx* G = a.GRc + (size_t)r * bb;
        for (int idx = threadIdx.x; idx < b * b; idx += 256) {
            const int i = idx / b, j = idx % b;
            cplx v = cmake(0.0, 0.0);
            for (int k = 0; k < b; k++) cfma(v, gl[i * b + k], G[k * b + j]);
            tmp[i * 33 + j] = v;
        }
        __syncthreads();
        double acc = 0.0;
        for (int idx = threadIdx.x; idx < b * b; idx += 256) {
            const int i = idx / b, j = idx % b;
            cplx v = cmake(0.0, 0.0);
            for (int k = 0; k < b; k++) cfma(v, tmp[i * 33 + k], gr[k * b + j]);
            const cplx g = G[idx];
            acc += v.x * g.x + v.y * g.y;
        }
        const double t = block_sum(acc);
        if (threadIdx.x == 0) a.trans[r] = t;
        return;
    }
    r -= a.n_trans;
    if (r < a.n_bond) { bond_current_body(r % (n - 1), r / (n - 1), n, b, a.Hu, a.Su, a.kidx, a.energy, a.GLu, a.bond); return; }
    r -= a.n_bond;
    contact_current_body(r & 1, r >> 1, n, b, a.sLl, a.sLg, a.sRl, a.sRg, a.GLd, a.GGd, a.contact);
}

}  // namespace

extern "C" int negf_observables(negf_ctx* ctx, const negf_problem* p,
                                const negf_c128* GR_diag, const negf_c128* GR_upper, const negf_c128* GR_lower,
                                const negf_c128* GR_corner, const negf_c128* GL_diag, const negf_c128* GL_upper,
                                const negf_c128* GG_diag, const negf_c128* gamma_L, const negf_c128* gamma_R,
                                const negf_c128* sigma_lesser_L, const negf_c128* sigma_greater_L,
                                const negf_c128* sigma_lesser_R, const negf_c128* sigma_greater_R,
                                const double* weights, double* density, double* ldos, double* transmission,
                                double* bond_current, double* contact_current) {
    if (!ctx || !p || p->n_blocks < 1 || p->block_size < 1 || p->n_energy < 1) return NEGF_EINVAL;
    const int n = p->n_blocks, b = p->block_size, ne = p->n_energy;
    const size_t bb = (size_t)b * b;
    const bool hasS = p->S_diag != nullptr;
    if (ne > 65535) return NEGF_EUNSUPPORTED;
    ProfScope _ps(ctx, NEGF_PROF_OBSERVABLES);
    if (p->n_k > 1 && !p->k_index) return NEGF_EINVAL;
    const int* kidx = p->n_k > 1 ? p->k_index : nullptr;        // k-point batching: S, H of the entry's own device
    if (fused_small_regime(ctx, b, ne)) {
        // resident small-block regime: every requested observable in one launch (argument checks as below)
        if (ldos && (!GR_diag || (hasS && n > 1 && (!GR_upper || !GR_lower || !p->S_upper)))) return NEGF_EINVAL;
        if (density && (!GL_diag || !weights || (hasS && n > 1 && (!GL_upper || !p->S_upper)))) return NEGF_EINVAL;
        if (transmission && (!GR_corner || !gamma_L || !gamma_R)) return NEGF_EINVAL;
        if (bond_current && n > 1 && (!GL_upper || !p->H_upper)) return NEGF_EINVAL;
        if (contact_current && (!GL_diag || !GG_diag || !sigma_lesser_L || !sigma_greater_L || !sigma_lesser_R || !sigma_greater_R))
            return NEGF_EINVAL;
        ObsSmallArgs a;
        a.n = n; a.b = b; a.ne = ne;
        a.GRd = (const cplx*)GR_diag; a.GRu = (const cplx*)GR_upper; a.GRl = (const cplx*)GR_lower; a.GRc = (const cplx*)GR_corner;
        a.GLd = (const cplx*)GL_diag; a.GLu = (const cplx*)GL_upper; a.GGd = (const cplx*)GG_diag;
        a.gamL = (const cplx*)gamma_L; a.gamR = (const cplx*)gamma_R;
        a.sLl = (const cplx*)sigma_lesser_L; a.sLg = (const cplx*)sigma_greater_L;
        a.sRl = (const cplx*)sigma_lesser_R; a.sRg = (const cplx*)sigma_greater_R;
        a.Hu = (const cplx*)p->H_upper; a.Sd = (const cplx*)p->S_diag; a.Su = (const cplx*)p->S_upper;
        a.kidx = kidx; a.energy = p->energy; a.w = weights;
        a.density = density; a.ldos = ldos; a.trans = transmission; a.bond = bond_current; a.contact = contact_current;
        a.n_ldos = ldos ? n * ne : 0;
        a.n_dens = density ? (n * b + 7) / 8 : 0;
        a.n_trans = transmission ? ne : 0;
        a.n_bond = (bond_current && n > 1) ? (n - 1) * ne : 0;
        a.n_contact = contact_current ? 2 * ne : 0;
        const long long blocks = (long long)a.n_ldos + a.n_dens + a.n_trans + a.n_bond + a.n_contact;
        if (blocks == 0) return NEGF_OK;
        if (blocks > 0x7fffffffLL) return NEGF_EUNSUPPORTED;
        obs_small_kernel<<<(unsigned)blocks, 256, 0, ctx->stream>>>(a);
        NEGF_LAUNCH_CHECK(ctx);
        return NEGF_OK;
    }
    if (ldos) {
        if (!GR_diag || (hasS && n > 1 && (!GR_upper || !GR_lower || !p->S_upper))) return NEGF_EINVAL;
        ldos_kernel<<<dim3(n, ne), 256, 0, ctx->stream>>>(n, b, (const cplx*)GR_diag, (const cplx*)GR_upper,
                                                          (const cplx*)GR_lower, (const cplx*)p->S_diag,
                                                          (const cplx*)p->S_upper, kidx, ldos);
        NEGF_LAUNCH_CHECK(ctx);
    }
    if (density) {
        if (!GL_diag || !weights || (hasS && n > 1 && (!GL_upper || !p->S_upper))) return NEGF_EINVAL;
        long long threads = (long long)n * b * 32;
        density_rows_kernel<<<(unsigned)((threads + 255) / 256), 256, 0, ctx->stream>>>(
            n, b, ne, (const cplx*)GL_diag, (const cplx*)GL_upper, (const cplx*)p->S_diag, (const cplx*)p->S_upper,
            kidx, weights, density);
        NEGF_LAUNCH_CHECK(ctx);
        if (hasS && n > 1) {
            density_cols_kernel<<<(n * b + DC_ROWS - 1) / DC_ROWS, dim3(DC_ROWS, DC_SLICES), 0, ctx->stream>>>(n, b, ne, (const cplx*)GL_upper,
                                                                            (const cplx*)p->S_upper, kidx, weights, density);
            NEGF_LAUNCH_CHECK(ctx);
        }
    }
    if (transmission) {
        if (!GR_corner || !gamma_L || !gamma_R) return NEGF_EINVAL;
        if (!ctx->ws) return NEGF_ENOWORKSPACE;
        Workspace W = carve_workspace(ctx->ws, n, b, ne);
        if (W.bytes > ctx->ws_bytes) return NEGF_ENOWORKSPACE;
        const cplx one = cmake(1.0, 0.0), zero = cmake(0.0, 0.0);
        // T = Re Tr[Gamma_L G Gamma_R G^H] = Re sum (Gamma_L G Gamma_R)[r][c] conj(G[r][c])
        NEGF_TRY(zgemm_bb(ctx, 0, 0, b, one, (const cplx*)gamma_L, bb, (const cplx*)GR_corner, bb, zero, nullptr, 0,
                          W.T[9], bb, ne, nullptr));
        NEGF_TRY(zgemm_bb(ctx, 0, 0, b, one, W.T[9], bb, (const cplx*)gamma_R, bb, zero, nullptr, 0, W.T[10], bb, ne, nullptr));
        dot_conj_kernel<<<dim3(1, ne), 256, 0, ctx->stream>>>(b, W.T[10], bb, (const cplx*)GR_corner, bb, 1.0,
                                                             transmission, 1, 0, 0);
        NEGF_LAUNCH_CHECK(ctx);
    }
    if (bond_current && n > 1) {
        if (!GL_upper || !p->H_upper) return NEGF_EINVAL;
        bond_current_kernel<<<dim3(n - 1, ne), 256, 0, ctx->stream>>>(n, b, (const cplx*)p->H_upper,
                                                                      (const cplx*)p->S_upper, kidx, p->energy,
                                                                      (const cplx*)GL_upper, bond_current);
        NEGF_LAUNCH_CHECK(ctx);
    }
    if (contact_current) {
        if (!GL_diag || !GG_diag || !sigma_lesser_L || !sigma_greater_L || !sigma_lesser_R || !sigma_greater_R)
            return NEGF_EINVAL;
        contact_current_kernel<<<dim3(2, ne), 256, 0, ctx->stream>>>(
            n, b, (const cplx*)sigma_lesser_L, (const cplx*)sigma_greater_L, (const cplx*)sigma_lesser_R,
            (const cplx*)sigma_greater_R, (const cplx*)GL_diag, (const cplx*)GG_diag, contact_current);
        NEGF_LAUNCH_CHECK(ctx);
    }
    return NEGF_OK;
}
