// O(b^2) kernels around the GEMM / inverse building blocks: assembly of the blocks of
// A = z S - H - Sigma^R and B = Sigma^<>, the anti-Hermitian combinations of
// S5/S6, the Sancho-Rubio bookkeeping (reading R3) and the boundary
// Gamma / Sigma^<> (8(c-2)).  All batched over energies: blockIdx.y = energy.
#include "common.cuh"
#include "kernels.cuh"

namespace {

__global__ void combine_kernel(const __grid_constant__ CombineArgs a) {
    const int e = blockIdx.y;
    if (a.skip && a.skip[e]) return;
    const int b = a.b;
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= b * b) return;
    const int r = idx / b, c = idx % b;
    const int fi = blockIdx.z;
    const size_t src = (a.dagger ? c * b + r : idx);
    const size_t kk = a.kidx ? (size_t)a.kidx[e] : 0;
    cplx v = cmake(0.0, 0.0);
    if (a.use_z) {
        cplx z = cmake(a.energy[e], a.eta);
        if (a.S) {
            cplx s = a.S[src + (size_t)fi * a.fS + kk * a.kS];
            if (a.dagger) s = cconj(s);
            v = cmul(z, s);
        } else if (a.s_identity && r == c) {
            v = z;
        }
    }
    if (a.H) {
        cplx h = a.H[src + (size_t)fi * a.fH + kk * a.kH];
        if (a.dagger) h = cconj(h);
        v = csub(v, h);
    }
    for (int t = 0; t < 3; t++) {
        if (a.blk[t] && (a.nfam <= 1 || a.only[t] < 0 || a.only[t] == fi)) {
            cplx x = a.blk[t][(size_t)e * a.sblk[t] + (a.only[t] < 0 ? (size_t)fi * a.fblk[t] : 0) + idx];
            v.x = fma(a.coef, x.x, v.x); v.y = fma(a.coef, x.y, v.y);
        }
    }
    if (a.scalar && r == c) {
        cplx x = a.scalar[e];
        v.x = fma(a.coef, x.x, v.x); v.y = fma(a.coef, x.y, v.y);
    }
    a.out[(size_t)e * a.sout + (size_t)fi * a.fout + idx] = v;
}

// C = Z + sign * (V - V^H)
__global__ void antiherm_add_kernel(int b, cplx* C, long long sC, const cplx* Z, long long sZ,
                                    const cplx* V, long long sV, double sign) {
    const int e = blockIdx.y;
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= b * b) return;
    const int r = idx / b, c = idx % b;
    cplx v = V[(size_t)e * sV + idx];
    cplx vt = V[(size_t)e * sV + c * b + r];
    cplx z = Z ? Z[(size_t)e * sZ + idx] : cmake(0.0, 0.0);
    C[(size_t)e * sC + idx] = cmake(z.x + sign * (v.x - vt.x), z.y + sign * (v.y + vt.y));
}

__global__ void sub_kernel(int b, cplx* C, long long sC, const cplx* A, long long sA, const cplx* B, long long sB) {
    const int e = blockIdx.y;
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= b * b) return;
    C[(size_t)e * sC + idx] = csub(A[(size_t)e * sA + idx], B[(size_t)e * sB + idx]);
}

__global__ void copy_kernel(size_t n, cplx* dst, long long sd, const cplx* src, long long ss, const int* skip) {
    const int e = blockIdx.y;
    if (skip && skip[e]) return;
    size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= n) return;
    dst[(size_t)e * sd + idx] = src[(size_t)e * ss + idx];
}

__global__ void fill_int_kernel(int* p, int n, int v) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) p[i] = v;
}
__global__ void max_int_kernel(int* dst, const int* src, int n) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) { int a = dst[i], s = src[i]; if (a == 0) dst[i] = s; }
}

// a_s -= lgu ; a_b -= ugl + lgu ; g = new a_b (the next doubling inverts g in place)
__global__ void sr_update_kernel(int b, cplx* a_s, cplx* a_b, cplx* g, const cplx* lgu, const cplx* ugl,
                                 const int* skip) {
    const int e = blockIdx.y;
    if (skip && skip[e]) return;
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= b * b) return;
    size_t o = (size_t)e * b * b + idx;
    cplx x = lgu[o], y = ugl[o];
    cplx s = a_s[o], d = a_b[o];
    a_s[o] = csub(s, x);
    d = cmake(d.x - x.x - y.x, d.y - x.y - y.y);
    a_b[o] = d; g[o] = d;
}

// update + norms + convergence test of one doubling in ONE launch.  gridDim.x (8 ... SR_SPLIT_MAX) CTAs per
// entry (the kernel is latency-bound per thread, not bandwidth-bound); the partial sums of squares
// go to acc[entry][SR_SPLIT_MAX][2] and the CTA that arrives last (ticket counter) adds them in a
// fixed order (deterministic) and takes the decision.
constexpr int SR_SPLIT_MAX = 128;     // sizes Workspace::acc (workspace.cuh)
__global__ void __launch_bounds__(256) sr_step_kernel(int b, cplx* a_s, cplx* a_b, cplx* g, const cplx* lgu,
                                                      const cplx* ugl, const cplx* un, const cplx* ln,
                                                      const double* ref, double tol, int* done, int* iters, int it,
                                                      double* acc, unsigned* ticket, const int* it_dev) {
    const int e = blockIdx.y;
    pdl_wait();                               // programmatic dependent launch (common.cuh)
    pdl_trigger();
    if (done[e]) return;
    if (it_dev) it += *it_dev;
    __shared__ double su[8], sl[8];
    const size_t o = (size_t)e * b * b;
    double au = 0.0, al = 0.0;
    const int split = gridDim.x;
    for (int i = blockIdx.x * 256 + threadIdx.x; i < b * b; i += 256 * split) {
        cplx x = lgu[o + i], y = ugl[o + i], s = a_s[o + i], d = a_b[o + i], u = un[o + i], l = ln[o + i];
        a_s[o + i] = csub(s, x);
        d = cmake(d.x - x.x - y.x, d.y - x.y - y.y);
        a_b[o + i] = d; g[o + i] = d;
        au += u.x * u.x + u.y * u.y;
        al += l.x * l.x + l.y * l.y;
    }
    for (int q = 16; q > 0; q >>= 1) {
        au += __shfl_down_sync(0xffffffffu, au, q);
        al += __shfl_down_sync(0xffffffffu, al, q);
    }
    if ((threadIdx.x & 31) == 0) { su[threadIdx.x >> 5] = au; sl[threadIdx.x >> 5] = al; }
    __syncthreads();
    if (threadIdx.x == 0) {
        au = 0.0; al = 0.0;
        for (int w = 0; w < 8; w++) { au += su[w]; al += sl[w]; }
        volatile double* slot = acc + (size_t)e * 2 * SR_SPLIT_MAX;
        slot[2 * blockIdx.x] = au; slot[2 * blockIdx.x + 1] = al;
        __threadfence();
        if (atomicAdd(&ticket[e], 1u) == (unsigned)split - 1u) {       // last CTA of this entry: fixed summation order
            __threadfence();
            double tu = 0.0, tl = 0.0;
            for (int q = 0; q < split; q++) { tu += slot[2 * q]; tl += slot[2 * q + 1]; }
            iters[e] = it + 1;
            if (sqrt(tu) + sqrt(tl) <= tol * ref[e]) done[e] = 1;
            ticket[e] = 0u;
        }
    }
}

// ||u||_F + ||l||_F per energy.  mode 0: ref[e] = value.  mode 1: convergence test (reading R3).
__global__ void sr_norm_kernel(int b, const cplx* u, const cplx* l, double* ref, double tol, int* done,
                               int* iters, int it, int mode) {
    const int e = blockIdx.x;
    if (mode == 1 && done[e]) return;
    __shared__ double su[32], sl[32];
    double au = 0.0, al = 0.0;
    const cplx* pu = u + (size_t)e * b * b;
    const cplx* pl = l + (size_t)e * b * b;
    for (int i = threadIdx.x; i < b * b; i += blockDim.x) {
        cplx x = pu[i], y = pl[i];
        au += x.x * x.x + x.y * x.y;
        al += y.x * y.x + y.y * y.y;
    }
    for (int o = 16; o > 0; o >>= 1) {
        au += __shfl_down_sync(0xffffffffu, au, o);
        al += __shfl_down_sync(0xffffffffu, al, o);
    }
    if ((threadIdx.x & 31) == 0) { su[threadIdx.x >> 5] = au; sl[threadIdx.x >> 5] = al; }
    __syncthreads();
    if (threadIdx.x == 0) {
        au = 0.0; al = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); w++) { au += su[w]; al += sl[w]; }
        double v = sqrt(au) + sqrt(al);
        if (mode == 0) ref[e] = v;
        else {
            iters[e] = it + 1;
            if (v <= tol * ref[e]) done[e] = 1;
        }
    }
}

// Gamma = i (Sigma - Sigma^H); f = fermi(E); Sigma^< = i f Gamma; Sigma^> = -i (1-f) Gamma
__global__ void obc_finalize_kernel(int b, const cplx* sigma, const double* energy, double mu, double kT,
                                    cplx* gamma, cplx* sl, cplx* sg, double* fermi) {
    const int e = blockIdx.y;
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    double x = (energy[e] - mu) / kT, f;
    if (x > 0) { double ex = exp(-x); f = ex / (1.0 + ex); } else { f = 1.0 / (1.0 + exp(x)); }
    if (idx == 0 && fermi) fermi[e] = f;
    if (idx >= b * b) return;
    const int r = idx / b, c = idx % b;
    size_t o = (size_t)e * b * b;
    cplx s = sigma[o + idx], st = sigma[o + c * b + r];
    // Sigma - Sigma^H = (s.x - st.x) + i (s.y + st.y) ;  times i
    cplx g = cmake(-(s.y + st.y), s.x - st.x);
    if (gamma) gamma[o + idx] = g;
    if (sl) sl[o + idx] = cmake(-f * g.y, f * g.x);                       // i f g
    if (sg) sg[o + idx] = cmake((1.0 - f) * g.y, -(1.0 - f) * g.x);       // -i (1-f) g
}

__global__ void obc_status_kernel(int ne, const int* done, const int* sing, const int* it_in, int* status,
                                  int* iters) {
    int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e < ne) { status[e] = sing[e] ? sing[e] : (done[e] ? 0 : -1); iters[e] = it_in[e]; }
}

// loop condition of the decimation WHILE graph: `step` more doublings while any entry is active
__global__ void sr_cond_kernel(cudaGraphConditionalHandle h, int nb, const int* done, int* it_dev, int max_iter, int step) {
    __shared__ int any;
    if (threadIdx.x == 0) any = 0;
    __syncthreads();
    for (int e = threadIdx.x; e < nb; e += blockDim.x) if (!done[e]) any = 1;
    __syncthreads();
    if (threadIdx.x == 0) {
        const int it = *it_dev + step;
        *it_dev = it;
        cudaGraphSetConditional(h, (any && it < max_iter) ? 1u : 0u);
    }
}

inline dim3 grid2(int b, int batch) { return dim3((b * b + 255) / 256, batch); }

}  // namespace

int ew_combine(negf_ctx* ctx, const CombineArgs& a, int batch) {
    ProfScope _ps(ctx, NEGF_PROF_ELEMENTWISE);
    dim3 grid = grid2(a.b, batch);
    grid.z = a.nfam > 1 ? a.nfam : 1;
    combine_kernel<<<grid, 256, 0, ctx->stream>>>(a);
    NEGF_LAUNCH_CHECK(ctx);
    return NEGF_OK;
}
int ew_antiherm_add(negf_ctx* ctx, int b, int batch, cplx* C, long long sC, const cplx* Z, long long sZ,
                    const cplx* V, long long sV, double sign) {
    ProfScope _ps(ctx, NEGF_PROF_ELEMENTWISE);
    antiherm_add_kernel<<<grid2(b, batch), 256, 0, ctx->stream>>>(b, C, sC, Z, sZ, V, sV, sign);
    NEGF_LAUNCH_CHECK(ctx);
    return NEGF_OK;
}
int ew_sub(negf_ctx* ctx, int b, int batch, cplx* C, long long sC, const cplx* A, long long sA,
           const cplx* B, long long sB) {
    ProfScope _ps(ctx, NEGF_PROF_ELEMENTWISE);
    sub_kernel<<<grid2(b, batch), 256, 0, ctx->stream>>>(b, C, sC, A, sA, B, sB);
    NEGF_LAUNCH_CHECK(ctx);
    return NEGF_OK;
}
int ew_copy(negf_ctx* ctx, size_t n, int batch, cplx* dst, long long sd, const cplx* src, long long ss,
            const int* skip) {
    ProfScope _ps(ctx, NEGF_PROF_ELEMENTWISE);
    copy_kernel<<<dim3((unsigned)((n + 255) / 256), batch), 256, 0, ctx->stream>>>(n, dst, sd, src, ss, skip);
    NEGF_LAUNCH_CHECK(ctx);
    return NEGF_OK;
}
int ew_fill_int(negf_ctx* ctx, int* p, int n, int v) {
    ProfScope _ps(ctx, NEGF_PROF_ELEMENTWISE);
    fill_int_kernel<<<(n + 255) / 256, 256, 0, ctx->stream>>>(p, n, v);
    NEGF_LAUNCH_CHECK(ctx);
    return NEGF_OK;
}
int ew_max_int(negf_ctx* ctx, int* dst, const int* src, int n) {
    ProfScope _ps(ctx, NEGF_PROF_ELEMENTWISE);
    max_int_kernel<<<(n + 255) / 256, 256, 0, ctx->stream>>>(dst, src, n);
    NEGF_LAUNCH_CHECK(ctx);
    return NEGF_OK;
}
int ew_sr_step(negf_ctx* ctx, int b, int batch, cplx* a_s, cplx* a_b, cplx* g, const cplx* lgu, const cplx* ugl,
               const cplx* un, const cplx* ln, const double* ref, double tol, int* done, int* iters, int it,
               double* acc, unsigned* ticket, const int* it_dev) {
    ProfScope _ps(ctx, NEGF_PROF_ELEMENTWISE);
    // one CTA per 16 K elements, at least 8 (the kernel is latency-bound per thread at small b), at most 128
    const int split = max(8, min(SR_SPLIT_MAX, (b * b + 16383) / 16384));
    NEGF_CUDA_CHECK(ctx, launch_chain(ctx, sr_step_kernel, dim3(split, batch), dim3(256), 0, b, a_s, a_b, g, lgu, ugl, un, ln, ref, tol,
                                      done, iters, it, acc, ticket, it_dev));
    NEGF_LAUNCH_CHECK(ctx);
    return NEGF_OK;
}
int ew_sr_cond(negf_ctx* ctx, cudaGraphConditionalHandle h, int nb, const int* done, int* it_dev, int max_iter, int step) {
    sr_cond_kernel<<<1, 128, 0, ctx->stream>>>(h, nb, done, it_dev, max_iter, step);
    NEGF_LAUNCH_CHECK(ctx);
    return NEGF_OK;
}
int ew_sr_update(negf_ctx* ctx, int b, int batch, cplx* a_s, cplx* a_b, cplx* g, const cplx* lgu,
                 const cplx* ugl, const int* skip) {
    ProfScope _ps(ctx, NEGF_PROF_ELEMENTWISE);
    sr_update_kernel<<<grid2(b, batch), 256, 0, ctx->stream>>>(b, a_s, a_b, g, lgu, ugl, skip);
    NEGF_LAUNCH_CHECK(ctx);
    return NEGF_OK;
}
int ew_sr_norm(negf_ctx* ctx, int b, int batch, const cplx* u, const cplx* l, double* ref, double tol,
               int* done, int* iters, int it, int mode) {
    ProfScope _ps(ctx, NEGF_PROF_ELEMENTWISE);
    sr_norm_kernel<<<batch, 256, 0, ctx->stream>>>(b, u, l, ref, tol, done, iters, it, mode);
    NEGF_LAUNCH_CHECK(ctx);
    return NEGF_OK;
}
int ew_obc_finalize(negf_ctx* ctx, int b, int batch, const cplx* sigma, const double* energy, double mu,
                    double kT, cplx* gamma, cplx* sl, cplx* sg, double* fermi) {
    ProfScope _ps(ctx, NEGF_PROF_ELEMENTWISE);
    obc_finalize_kernel<<<grid2(b, batch), 256, 0, ctx->stream>>>(b, sigma, energy, mu, kT, gamma, sl, sg, fermi);
    NEGF_LAUNCH_CHECK(ctx);
    return NEGF_OK;
}
int ew_obc_status(negf_ctx* ctx, int ne, const int* done, const int* sing, const int* it_in, int* status, int* iters) {
    ProfScope _ps(ctx, NEGF_PROF_ELEMENTWISE);
    obc_status_kernel<<<(ne + 255) / 256, 256, 0, ctx->stream>>>(ne, done, sing, it_in, status, iters);
    NEGF_LAUNCH_CHECK(ctx);
    return NEGF_OK;
}
