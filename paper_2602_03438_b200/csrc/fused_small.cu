// Resident small-block regime (b <= 32): the WHOLE chain of one energy in ONE CTA (SURVEY.md section 7 step 3,
// BASELINE.json north_star "the energy-batch scheduler that packs small blocks of many energies into one launch").
//
// "Eqs. (1) and (2) can be solved with the so-called recursive Green's function (RGF) algorithm, which is
// sequential in essence": at b <= 32 every step of the chain is a few microseconds of arithmetic, and
// as separate batched launches the path is pure launch latency (configs[0]: 305 launches, 0.76 ms for 15 MFLOP).
// Here one thread block walks the chain of its energy with every operand in shared memory:
//   fused_obc_kernel   S2: one CTA per (lead, energy) runs the complete Sancho-Rubio doubling loop -
//                      inverse, six products, update, norms, stopping rule (reading R3) - and the boundary blocks
//                      Sigma^R, Gamma, Sigma^<, Sigma^>; a converged entry simply leaves the loop;
//   fused_ret_kernel   S1+S3+S4: one CTA per energy, forward and backward retarded sweeps, the blocks of
//                      A assembled on the fly from H, S, z and Sigma^R; g_i, X_i, Y_i go to the workspace in the
//                      one-sided layout of rgf.cu (retained sweep state), the selected G^R blocks to the outputs;
//   fused_lg_kernel    S5+S6: one CTA per (energy, < or >), textbook forward recursion and the compact backward form.
// Building blocks inside the CTA: complex b x b x b products on the FP64 pipe out of shared memory (DFMA; at these
// sizes a product is 100-400 ns and latency-, not pipe-bound) and a warp-resident Gauss-Jordan inverse with
// implicit threshold pivoting (lane = row, the row in registers, the column being eliminated always in register 0
// with the row rotated by one register per step - the scheme of zinv_rows.cu for one warp).
// Same arithmetic definitions as the batched path (obc.cu, rgf.cu); results agree to rounding, not to the bit.
#include "common.cuh"
#include "fused_small.cuh"

namespace {

constexpr int FNT = 256;                       // threads per CTA
constexpr unsigned FULLM = 0xffffffffu;

template <int FB> struct Mat { static constexpr int LD = FB + 1; static constexpr int SZ = FB * (FB + 1); };

__device__ __forceinline__ cplx f_recip(cplx a) {
    const double x = fma(a.x, a.x, a.y * a.y);
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    double e = fma(-x, r, 1.0);
    r = fma(r, e, r);
    e = fma(-x, r, 1.0);
    r = fma(r, e, r);
    return cmake(a.x * r, -a.y * r);
}

// C = alpha * op(A) * op(B) + beta * D  (b x b, all in shared memory, leading dimension FB + 1; D may be C or
// null).  Thread t owns column c = t % FB of the rows r = t / FB + j * (FNT / FB).  Two accumulator sets (even / odd
// k) halve the dependent DFMA chain, which is what a product costs at these sizes.  ALIAS: C is also an operand
// (one more barrier between the last read and the first write).  Ends with a block barrier.
template <int FB, int OPA, int OPB, bool ALIAS = false>
__device__ __forceinline__ void f_gemm(cplx* C, const cplx* A, const cplx* B, int b, cplx alpha, cplx beta, const cplx* D) {
    constexpr int LD = Mat<FB>::LD, RS = FNT / FB, NR = FB / RS;
    const int c = threadIdx.x % FB, r0 = threadIdx.x / FB;
    cplx acc[NR], acc2[NR];
#pragma unroll
    for (int j = 0; j < NR; j++) { acc[j] = cmake(0.0, 0.0); acc2[j] = cmake(0.0, 0.0); }
    if (c < b) {
        int k = 0;
#pragma unroll 2
        for (; k + 1 < b; k += 2) {
            const cplx b0 = OPB ? cconj(B[c * LD + k]) : B[k * LD + c];
            const cplx b1 = OPB ? cconj(B[c * LD + k + 1]) : B[(k + 1) * LD + c];
#pragma unroll
            for (int j = 0; j < NR; j++) {
                const int r = r0 + j * RS;
                const cplx a0 = OPA ? cconj(A[k * LD + r]) : A[r * LD + k];
                const cplx a1 = OPA ? cconj(A[(k + 1) * LD + r]) : A[r * LD + k + 1];
                cfma(acc[j], a0, b0);
                cfma(acc2[j], a1, b1);
            }
        }
        if (k < b) {
            const cplx b0 = OPB ? cconj(B[c * LD + k]) : B[k * LD + c];
#pragma unroll
            for (int j = 0; j < NR; j++) {
                const int r = r0 + j * RS;
                cfma(acc[j], OPA ? cconj(A[k * LD + r]) : A[r * LD + k], b0);
            }
        }
    }
    if (ALIAS) __syncthreads();
    if (c < b) {
#pragma unroll
        for (int j = 0; j < NR; j++) {
            const int r = r0 + j * RS;
            if (r < b) {
                cplx v = cmul(alpha, cadd(acc[j], acc2[j]));
                if (D) cfma(v, beta, D[r * LD + c]);
                C[r * LD + c] = v;
            }
        }
    }
    __syncthreads();
}

// element-wise helpers over the b x b block (all threads), each ends with a barrier
template <int FB, class F>
__device__ __forceinline__ void f_each(int b, F f) {
    constexpr int LD = Mat<FB>::LD;
    for (int idx = threadIdx.x; idx < b * b; idx += FNT) { const int r = idx / b, c = idx % b; f(r, c, r * LD + c); }
    __syncthreads();
}
// In-place inverse of the b x b block M (shared memory) by warp 0: Gauss-Jordan with implicit threshold pivoting on
// the leading 32 bits of |re|+|im| (lowest row among equals).  The block is treated as FB x FB padded with the
// identity (padding rows pivot on padding columns).  `line` = FB complex of shared scratch.  Returns (to every
// thread, after a barrier) 0 or the 1-based column of the first zero pivot through *sing_out (shared int).
// One elimination step; (p, kmax) = pivot lane and key of the column in register 0 of x (found by the previous step).
// The next column is updated FIRST and its pivot search (redux + ballot) is issued before the other columns'
// updates, so that its latency hides under them; returns the next pivot in (p, kmax).
template <int FB>
__device__ __forceinline__ void f_search(const cplx v, bool used, int k, int b, int lane, int& p, unsigned& kmax) {
    const bool elig = !used && ((lane < b) == (k < b)) && lane < FB;
    unsigned key = 0u;
    if (elig) key = (unsigned)((unsigned long long)__double_as_longlong(cabs1(v)) >> 32) + 1u;
    kmax = __reduce_max_sync(FULLM, key);
    const unsigned bal = __ballot_sync(FULLM, elig && key == kmax);
    p = bal ? __ffs(bal) - 1 : 0;
}
template <int FB>
__device__ __forceinline__ void f_step(const cplx (&x)[FB], cplx (&y)[FB], bool& used, int& piv_of_col, int k, int b, int lane,
                                       cplx* line, int* sing, int& p, unsigned& kmax) {
    if (kmax <= 1u && k < b && lane == 0 && *sing == 0) *sing = k + 1;
    if (lane == p) {
#pragma unroll
        for (int c = 0; c < FB; c++) line[c] = x[c];
    }
    if (lane == k) piv_of_col = p;                   // lane k remembers the pivot row of column k
    __syncwarp();
    const cplx d = kmax <= 1u ? cmake(1.0, 0.0) : f_recip(line[0]);
    const bool isp = lane == p;
    const cplx m = cmul(x[0], d);
    if (isp) used = true;
    { cplx t = x[1]; if (isp) t = cmul(t, d); else cfms(t, m, line[1]); y[0] = t; }
    int pn; unsigned kn;
    f_search<FB>(y[0], used, k + 1, b, lane, pn, kn);
#pragma unroll
    for (int c = 2; c < FB; c++) { cplx t = x[c]; if (isp) t = cmul(t, d); else cfms(t, m, line[c]); y[c - 1] = t; }
    y[FB - 1] = isp ? d : cneg(m);
    p = pn; kmax = kn;
    __syncwarp();
}

// In-place inverse of the b x b block M (shared memory; `src` = where the matrix is read from, may be M) by warp 0:
// Gauss-Jordan with implicit threshold pivoting on the leading 32 bits of |re|+|im| (lowest row among equals).  The
// block is treated as FB x FB padded with the identity (padding rows pivot on padding columns).  `line` = FB complex
// of shared scratch, piv = 2 FB ints.  *sing (shared) = 0 or the 1-based column of the first zero pivot.
template <int FB>
__device__ __noinline__ void f_inverse(cplx* M, const cplx* src, int b, cplx* line, int* piv, int* sing) {
    constexpr int LD = Mat<FB>::LD;
    if (threadIdx.x == 0) *sing = 0;
    __syncthreads();
    if (threadIdx.x < 32) {
        const int lane = threadIdx.x;
        cplx x[FB], y[FB];
#pragma unroll
        for (int c = 0; c < FB; c++)
            x[c] = (lane < b && c < b) ? src[lane * LD + c] : cmake(lane == c ? 1.0 : 0.0, 0.0);
        bool used = false; int pk = 0, p; unsigned kmax;
        f_search<FB>(x[0], used, 0, b, lane, p, kmax);
#pragma unroll 1
        for (int k = 0; k < FB; k += 2) {
            f_step<FB>(x, y, used, pk, k, b, lane, line, sing, p, kmax);
            f_step<FB>(y, x, used, pk, k + 1, b, lane, line, sing, p, kmax);
        }
        // lane i holds B[i][j] = X[i][piv[j]], X = Pi A^-1 (zinv.cu): A^-1[pinv[i]][piv[j]] = B[i][j]
        if (lane < FB) piv[lane] = pk;
        __syncwarp();
        if (lane < FB) piv[FB + piv[lane]] = lane;                  // pinv
        __syncwarp();
        if (lane < b) {
            const int dr = piv[FB + lane];
#pragma unroll
            for (int c = 0; c < FB; c++)
                if (c < b) M[dr * LD + piv[c]] = x[c];
        }
    }
    __syncthreads();
}

// One Newton step on an inverse, X <- X + X (I - A X) (tmp = scratch block).  The doubling is conditioning-limited
// (hazard H2) and every g = a_b^-1 feeds six products: a Gauss-Jordan inverse measured 2-6x the error of an LU-based
// one on near-singular symmetric lead blocks (numpy emulation of both in the doubling); the
// step brings it to the LU level for two products of 0.2 us.
template <int FB>
__device__ __forceinline__ void f_refine(cplx* X, const cplx* A, cplx* tmp, int b) {
    constexpr int LD = Mat<FB>::LD;
    f_gemm<FB, 0, 0>(tmp, A, X, b, cmake(-1.0, 0.0), cmake(0.0, 0.0), nullptr);
    for (int i = threadIdx.x; i < b; i += FNT) tmp[i * LD + i].x += 1.0;
    __syncthreads();
    f_gemm<FB, 0, 0, true>(X, X, tmp, b, cmake(1.0, 0.0), cmake(1.0, 0.0), X);
}

// ---- global <-> shared block copies (b x b, global leading dimension b), each ends with a barrier ----------------
template <int FB>
__device__ __forceinline__ void g2s(cplx* S, const cplx* g, int b) {
    constexpr int LD = Mat<FB>::LD;
    for (int idx = threadIdx.x; idx < b * b; idx += FNT) S[(idx / b) * LD + idx % b] = g[idx];
    __syncthreads();
}
template <int FB>
__device__ __forceinline__ void s2g(cplx* g, const cplx* S, int b) {
    constexpr int LD = Mat<FB>::LD;
    if (g) for (int idx = threadIdx.x; idx < b * b; idx += FNT) g[idx] = S[(idx / b) * LD + idx % b];
    __syncthreads();
}
template <int FB>
__device__ __forceinline__ void s2s(cplx* D, const cplx* S, int b) {
    constexpr int LD = Mat<FB>::LD;
    for (int idx = threadIdx.x; idx < b * b; idx += FNT) { const int o = (idx / b) * LD + idx % b; D[o] = S[o]; }
    __syncthreads();
}

// ---- blocks of A = z S - H - Sigma^R for batch entry e, assembled into shared memory --------------
// which: 0 diagonal block i, 1 upper block A_{i,i+1}, 2 lower block A_{i+1,i}
template <int FB>
__device__ __forceinline__ void load_A(cplx* S, const FusedProblem& P, int e, int i, int which) {
    constexpr int LD = Mat<FB>::LD;
    const int b = P.b, n = P.n;
    const size_t bb = (size_t)b * b;
    const cplx z = cmake(P.energy[e], P.eta);
    const size_t kk = P.kidx ? (size_t)P.kidx[e] : 0;
    const cplx* H = which == 0 ? P.Hd + (kk * n + i) * bb : P.Hu + (kk * (n - 1) + i) * bb;
    const cplx* Sm = which == 0 ? (P.Sd ? P.Sd + (kk * n + i) * bb : nullptr) : (P.Su ? P.Su + (kk * (n - 1) + i) * bb : nullptr);
    const cplx* sg = nullptr;                       // dense Sigma^R_S block of this entry
    if (P.sr_kind == NEGF_SIGMA_BT)
        sg = which == 0 ? P.sr_diag + ((size_t)e * n + i) * bb
                        : (which == 1 ? P.sr_upper : P.sr_lower) + ((size_t)e * (n - 1) + i) * bb;
    const cplx* bnd = nullptr;
    if (which == 0 && i == 0 && P.sr_left) bnd = P.sr_left + (size_t)e * bb;
    const cplx* bnd2 = (which == 0 && i == n - 1 && P.sr_right) ? P.sr_right + (size_t)e * bb : nullptr;
    const cplx sc = (which == 0 && P.sr_kind == NEGF_SIGMA_SCALAR) ? P.sr_scalar[e] : cmake(0.0, 0.0);
    for (int idx = threadIdx.x; idx < b * b; idx += FNT) {
        const int r = idx / b, c = idx % b;
        const int src = which == 2 ? c * b + r : idx;            // lower block = dagger of the upper arrays of H and S
        cplx h = H[src], v;
        if (which == 2) h = cconj(h);
        if (Sm) { cplx s = Sm[src]; if (which == 2) s = cconj(s); v = cmul(z, s); }
        else v = (which == 0 && r == c) ? z : cmake(0.0, 0.0);
        v = csub(v, h);
        if (sg) v = csub(v, sg[idx]);
        if (bnd) v = csub(v, bnd[idx]);
        if (bnd2) v = csub(v, bnd2[idx]);
        if (r == c) v = csub(v, sc);
        S[r * LD + c] = v;
    }
    __syncthreads();
}

// ||U||_F + ||L||_F of two blocks: one block reduction in a fixed order; result to every thread
template <int FB>
__device__ __forceinline__ double f_norm_pair(const cplx* U, const cplx* L, int b, double* red) {
    constexpr int LD = Mat<FB>::LD;
    double a = 0.0, c = 0.0;
    for (int idx = threadIdx.x; idx < b * b; idx += FNT) {
        const int o = (idx / b) * LD + idx % b;
        const cplx v = U[o], w = L[o];
        a += v.x * v.x + v.y * v.y; c += w.x * w.x + w.y * w.y;
    }
    for (int o = 16; o > 0; o >>= 1) { a += __shfl_down_sync(FULLM, a, o); c += __shfl_down_sync(FULLM, c, o); }
    if ((threadIdx.x & 31) == 0) { red[threadIdx.x >> 5] = a; red[8 + (threadIdx.x >> 5)] = c; }
    __syncthreads();
    double ta = 0.0, tc = 0.0;
    for (int w = 0; w < FNT / 32; w++) { ta += red[w]; tc += red[8 + w]; }
    __syncthreads();
    return sqrt(ta) + sqrt(tc);
}

// ---------------------------------------------------------------------------------------------------------------------
// S2: Sancho-Rubio decimation, one CTA per (lead, energy)
// ---------------------------------------------------------------------------------------------------------------------
template <int FB>
__global__ void __launch_bounds__(FNT, 1) fused_obc_kernel(const FusedObcArgs a) {
    constexpr int LD = Mat<FB>::LD, SZ = Mat<FB>::SZ;
    extern __shared__ __align__(16) unsigned char fsm[];
    cplx* m = reinterpret_cast<cplx*>(fsm);
    cplx *a_s = m, *a_b = m + SZ, *g = m + 2 * SZ, *u = m + 3 * SZ, *l = m + 4 * SZ, *un = m + 5 * SZ, *ln = m + 6 * SZ,
         *gu = m + 7 * SZ, *gl = m + 8 * SZ, *t = m + 9 * SZ, *U0 = m + 10 * SZ, *L0 = m + 11 * SZ;
    cplx* line = m + 12 * SZ;                                       // [FB]
    double* red = reinterpret_cast<double*>(line + FB);            // [16]
    int* piv = reinterpret_cast<int*>(red + 16);                   // [2 FB]
    int* sing = piv + 2 * FB;
    const int b = a.b, ne = a.ne;
    const int s = blockIdx.x / ne, e = blockIdx.x % ne;             // lead slot, energy
    const FusedLead& L = a.lead[s];
    const size_t bb = (size_t)b * b;
    const cplx z = cmake(a.energy[e], a.eta);
    const size_t kk = a.kidx ? (size_t)a.kidx[e] : 0;
    // lead blocks a_d, a_u, a_l; a right lead stores (u, l) exchanged and runs the left-lead recursion (obc.cu)
    cplx* Uq = L.side == 0 ? U0 : L0;                               // receives a_u
    cplx* Lq = L.side == 0 ? L0 : U0;                               // receives a_l
    for (int idx = threadIdx.x; idx < b * b; idx += FNT) {
        const int r = idx / b, c = idx % b, o = r * LD + c;
        cplx v = L.Sd ? cmul(z, L.Sd[kk * L.kd + idx]) : (r == c ? z : cmake(0.0, 0.0));
        v = csub(v, L.Hd[kk * L.kd + idx]);
        a_s[o] = v; a_b[o] = v;
        cplx up = L.Su ? cmul(z, L.Su[kk * L.ku + idx]) : cmake(0.0, 0.0);
        Uq[o] = csub(up, L.Hu[kk * L.ku + idx]);
        const int tr = c * b + r;
        cplx lo = L.Su ? cmul(z, cconj(L.Su[kk * L.ku + tr])) : cmake(0.0, 0.0);
        Lq[o] = csub(lo, cconj(L.Hu[kk * L.ku + tr]));
    }
    __syncthreads();
    s2s<FB>(u, U0, b); s2s<FB>(l, L0, b);
    const double ref = f_norm_pair<FB>(U0, L0, b, red);
    const cplx one = cmake(1.0, 0.0), mone = cmake(-1.0, 0.0), zero = cmake(0.0, 0.0);
    int iters = 0, done = 0, sing_code = 0;
    for (int it = 0; it < a.max_iter; it++) {
        f_inverse<FB>(g, a_b, b, line, piv, sing);                  // g = a_b^-1
        if (*sing && !sing_code) sing_code = it + 1;
        f_refine<FB>(g, a_b, gu, b);
        f_gemm<FB, 0, 0>(gu, g, u, b, one, zero, nullptr);          // g u
        f_gemm<FB, 0, 0>(gl, g, l, b, one, zero, nullptr);          // g l
        f_gemm<FB, 0, 0>(t, l, gu, b, one, zero, nullptr);          // l g u
        f_each<FB>(b, [&](int, int, int o) { a_s[o] = csub(a_s[o], t[o]); a_b[o] = csub(a_b[o], t[o]); });
        f_gemm<FB, 0, 0>(a_b, u, gl, b, mone, one, a_b);            // a_b -= u g l
        f_gemm<FB, 0, 0>(un, u, gu, b, mone, zero, nullptr);        // u <- -u g u
        f_gemm<FB, 0, 0>(ln, l, gl, b, mone, zero, nullptr);        // l <- -l g l
        cplx* sw = u; u = un; un = sw; sw = l; l = ln; ln = sw;
        iters = it + 1;
        const double nrm = f_norm_pair<FB>(u, l, b, red);
        if (nrm <= a.tol * ref) { done = 1; break; }                // reading R3 (uniform over the CTA)
    }
    s2s<FB>(g, a_s, b);
    f_inverse<FB>(a_s, a_s, b, line, piv, sing);                    // g_s = a_s^-1
    if (*sing && !sing_code) sing_code = a.max_iter + 1;
    f_refine<FB>(a_s, g, gu, b);
    f_gemm<FB, 0, 0>(gu, a_s, U0, b, one, zero, nullptr);
    f_gemm<FB, 0, 0>(t, L0, gu, b, one, zero, nullptr);             // Sigma^R (exchanged storage: a_u g_s a_l for a right lead)
    // outputs
    const double xx = (a.energy[e] - L.mu) / a.kT;
    double f;
    if (xx > 0) { const double ex = exp(-xx); f = ex / (1.0 + ex); } else { f = 1.0 / (1.0 + exp(xx)); }
    const size_t off = (size_t)e * bb;
    for (int idx = threadIdx.x; idx < b * b; idx += FNT) {
        const int r = idx / b, c = idx % b;
        const cplx sv = t[r * LD + c], st = t[c * LD + r];
        const cplx gm = cmake(-(sv.y + st.y), sv.x - st.x);          // i (Sigma - Sigma^H)
        L.sigma_r[off + idx] = sv;
        if (L.gamma) L.gamma[off + idx] = gm;
        if (L.sigma_lesser) L.sigma_lesser[off + idx] = cmake(-f * gm.y, f * gm.x);
        if (L.sigma_greater) L.sigma_greater[off + idx] = cmake((1.0 - f) * gm.y, -(1.0 - f) * gm.x);
        if (L.g_surface) L.g_surface[off + idx] = a_s[r * LD + c];
    }
    if (threadIdx.x == 0) {
        if (L.fermi) L.fermi[e] = f;
        L.iters[e] = iters;
        L.status[e] = sing_code ? sing_code : (done ? 0 : -1);
    }
}

// ---------------------------------------------------------------------------------------------------------------------
// S1 + S3 + S4: retarded sweeps, one CTA per energy
// ---------------------------------------------------------------------------------------------------------------------
template <int FB>
__global__ void __launch_bounds__(FNT, 1) fused_ret_kernel(const FusedProblem P, const FusedRetOut o) {
    constexpr int SZ = Mat<FB>::SZ;
    extern __shared__ __align__(16) unsigned char fsm[];
    cplx* m = reinterpret_cast<cplx*>(fsm);
    cplx *M = m, *gp = m + SZ, *A1 = m + 2 * SZ, *Y = m + 3 * SZ, *X = m + 4 * SZ, *G = m + 5 * SZ, *T = m + 6 * SZ,
         *col = m + 7 * SZ, *Gn = m + 8 * SZ;
    cplx* line = m + 9 * SZ;
    double* red = reinterpret_cast<double*>(line + FB);
    int* piv = reinterpret_cast<int*>(red + 16);
    int* sing = piv + 2 * FB;
    const int b = P.b, n = P.n, e = blockIdx.x;
    const size_t bb = (size_t)b * b;
    cplx* Wg = o.g + (size_t)e * n * bb;
    cplx* WX = o.X + (size_t)e * (n - 1) * bb;
    cplx* WY = o.Y + (size_t)e * (n - 1) * bb;
    const cplx one = cmake(1.0, 0.0), mone = cmake(-1.0, 0.0), zero = cmake(0.0, 0.0);
    int code = 0;
    // S3: g_0 = A_00^-1; Y_{i-1} = A_{i,i-1} g_{i-1}; g_i = (A_ii - Y_{i-1} A_{i-1,i})^-1
    for (int i = 0; i < n; i++) {
        load_A<FB>(M, P, e, i, 0);
        if (i > 0) {
            load_A<FB>(A1, P, e, i - 1, 2);                               // A_{i,i-1}
            f_gemm<FB, 0, 0>(Y, A1, gp, b, one, zero, nullptr);
            s2g<FB>(WY + (size_t)(i - 1) * bb, Y, b);
            load_A<FB>(A1, P, e, i - 1, 1);                               // A_{i-1,i}
            f_gemm<FB, 0, 0>(M, Y, A1, b, mone, one, M);
        }
        f_inverse<FB>(M, M, b, line, piv, sing);
        if (*sing && !code) code = i + 1;
        s2g<FB>(Wg + (size_t)i * bb, M, b);
        cplx* sw = gp; gp = M; M = sw;                                    // g_{i} stays resident for the next step
    }
    // S4: G_{n-1,n-1} = g_{n-1}; X_i = g_i A_{i,i+1}; G_{i,i+1} = -X_i G_{i+1,i+1}; G_{i+1,i} = -G_{i+1,i+1} Y_i;
    //     G_ii = g_i - G_{i,i+1} Y_i; corner column G_{i,n-1} = -X_i G_{i+1,n-1}
    s2s<FB>(G, gp, b);
    s2g<FB>(o.GR_diag + ((size_t)e * n + n - 1) * bb, G, b);
    if (o.GR_corner) s2s<FB>(col, gp, b);
    for (int i = n - 2; i >= 0; i--) {
        g2s<FB>(gp, Wg + (size_t)i * bb, b);
        load_A<FB>(A1, P, e, i, 1);
        f_gemm<FB, 0, 0>(X, gp, A1, b, one, zero, nullptr);
        s2g<FB>(WX + (size_t)i * bb, X, b);
        g2s<FB>(Y, WY + (size_t)i * bb, b);
        f_gemm<FB, 0, 0>(T, X, G, b, mone, zero, nullptr);                // G_{i,i+1}
        s2g<FB>(o.GR_upper ? o.GR_upper + ((size_t)e * (n - 1) + i) * bb : nullptr, T, b);
        if (o.GR_lower) {
            f_gemm<FB, 0, 0>(Gn, G, Y, b, mone, zero, nullptr);           // G_{i+1,i}
            s2g<FB>(o.GR_lower + ((size_t)e * (n - 1) + i) * bb, Gn, b);
        }
        f_gemm<FB, 0, 0>(Gn, T, Y, b, mone, one, gp);                     // G_ii
        s2g<FB>(o.GR_diag + ((size_t)e * n + i) * bb, Gn, b);
        if (o.GR_corner) f_gemm<FB, 0, 0, true>(col, X, col, b, mone, zero, nullptr);
        cplx* sw = G; G = Gn; Gn = sw;
    }
    if (o.GR_corner) s2g<FB>(o.GR_corner + (size_t)e * bb, col, b);
    if (threadIdx.x == 0 && code && o.info[e] == 0) o.info[e] = code;
}

// ---------------------------------------------------------------------------------------------------------------------
// S5 + S6: lesser / greater sweeps, one CTA per (energy, < or >)
// ---------------------------------------------------------------------------------------------------------------------
template <int FB>
__global__ void __launch_bounds__(FNT, 1) fused_lg_kernel(const FusedProblem P, const FusedLgArgs a) {
    constexpr int SZ = Mat<FB>::SZ;
    extern __shared__ __align__(16) unsigned char fsm[];
    cplx* m = reinterpret_cast<cplx*>(fsm);
    cplx *gx = m, *gi = m + SZ, *A1 = m + 2 * SZ, *Bm = m + 3 * SZ, *T = m + 4 * SZ, *T2 = m + 5 * SZ, *Yp = m + 6 * SZ,
         *X = m + 7 * SZ, *GX = m + 8 * SZ, *Q = m + 9 * SZ, *GR = m + 10 * SZ;
    const int b = P.b, n = P.n, e = blockIdx.x;
    const FusedLgOne& S = a.x[blockIdx.y];
    const size_t bb = (size_t)b * b;
    const cplx* Wg = a.g + (size_t)e * n * bb;
    const cplx* WX = a.X + (size_t)e * (n - 1) * bb;
    const cplx* WY = a.Y + (size_t)e * (n - 1) * bb;
    cplx* Wgx = S.gx + (size_t)e * n * bb;
    const cplx one = cmake(1.0, 0.0), mone = cmake(-1.0, 0.0), zero = cmake(0.0, 0.0);
    constexpr int LD = Mat<FB>::LD;
    // S5: g^x_0 = g_0 B_00 g_0^H; g^x_i = g_i [B_ii + A_{i,i-1} g^x_{i-1} A_{i,i-1}^H - (V - V^H)] g_i^H, V = Y_{i-1} B_{i-1,i}
    for (int i = 0; i < n; i++) {
        const cplx sc = S.kind == NEGF_SIGMA_SCALAR ? S.scalar[e] : cmake(0.0, 0.0);
        const cplx* sd = S.kind == NEGF_SIGMA_BT ? S.diag + ((size_t)e * n + i) * bb : nullptr;
        const cplx* bl = (i == 0 && S.left) ? S.left + (size_t)e * bb : nullptr;
        const cplx* br = (i == n - 1 && S.right) ? S.right + (size_t)e * bb : nullptr;
        f_each<FB>(b, [&](int r, int c, int oo) {
            const int idx = r * b + c;
            cplx v = r == c ? sc : cmake(0.0, 0.0);
            if (sd) v = cadd(v, sd[idx]);
            if (bl) v = cadd(v, bl[idx]);
            if (br) v = cadd(v, br[idx]);
            Bm[oo] = v;
        });
        if (i > 0) {
            load_A<FB>(A1, P, e, i - 1, 2);                               // A_{i,i-1}
            f_gemm<FB, 0, 0>(T, A1, gx, b, one, zero, nullptr);
            f_gemm<FB, 0, 1>(Bm, T, A1, b, one, one, Bm);                 // + A g^x A^H
            if (S.kind == NEGF_SIGMA_BT) {
                g2s<FB>(Yp, WY + (size_t)(i - 1) * bb, b);
                g2s<FB>(T2, S.upper + ((size_t)e * (n - 1) + i - 1) * bb, b);
                f_gemm<FB, 0, 0>(T, Yp, T2, b, one, zero, nullptr);       // V
                f_each<FB>(b, [&](int r, int c, int oo) {
                    const cplx v = T[oo], vt = T[c * LD + r];
                    Bm[oo] = cmake(Bm[oo].x - (v.x - vt.x), Bm[oo].y - (v.y + vt.y));     // - (V - V^H)
                });
            }
        }
        g2s<FB>(gi, Wg + (size_t)i * bb, b);
        f_gemm<FB, 0, 0>(T, gi, Bm, b, one, zero, nullptr);
        f_gemm<FB, 0, 1>(gx, T, gi, b, one, zero, nullptr);
        s2g<FB>(Wgx + (size_t)i * bb, gx, b);
    }
    // S6: G^x_{n-1,n-1} = g^x_{n-1};  T2 = -g^x_i A_{i+1,i}^H + g_i B_{i,i+1};  Q = T2 (G^R_{i+1,i+1})^H;
    //     G^x_{i,i+1} = Q - X_i G^x_{i+1,i+1};  G^x_ii = g^x_i - Q X_i^H + X_i (G^x_{i,i+1})^H
    s2s<FB>(GX, gx, b);
    s2g<FB>(S.GX_diag + ((size_t)e * n + n - 1) * bb, GX, b);
    for (int i = n - 2; i >= 0; i--) {
        g2s<FB>(gx, Wgx + (size_t)i * bb, b);
        load_A<FB>(A1, P, e, i, 2);                                       // A_{i+1,i}
        f_gemm<FB, 0, 1>(T2, gx, A1, b, mone, zero, nullptr);
        if (S.kind == NEGF_SIGMA_BT) {
            g2s<FB>(gi, Wg + (size_t)i * bb, b);
            g2s<FB>(T, S.upper + ((size_t)e * (n - 1) + i) * bb, b);
            f_gemm<FB, 0, 0>(T2, gi, T, b, one, one, T2);
        }
        g2s<FB>(GR, a.GR_diag + ((size_t)e * n + i + 1) * bb, b);
        f_gemm<FB, 0, 1>(Q, T2, GR, b, one, zero, nullptr);
        g2s<FB>(X, WX + (size_t)i * bb, b);
        f_gemm<FB, 0, 1>(gx, Q, X, b, mone, one, gx);                     // P_i = g^x_i - Q X^H
        f_gemm<FB, 0, 0>(Q, X, GX, b, mone, one, Q);                      // G^x_{i,i+1}
        s2g<FB>(S.GX_upper ? S.GX_upper + ((size_t)e * (n - 1) + i) * bb : nullptr, Q, b);
        f_gemm<FB, 0, 1>(GX, X, Q, b, one, one, gx);                      // G^x_ii
        s2g<FB>(S.GX_diag + ((size_t)e * n + i) * bb, GX, b);
    }
}

template <int FB> constexpr size_t fused_smem(int nmat) {
    return (size_t)nmat * Mat<FB>::SZ * sizeof(cplx) + FB * sizeof(cplx) + 16 * sizeof(double) + (2 * FB + 4) * sizeof(int);
}

}  // namespace

int fused_prepare(negf_ctx* ctx) {
    NEGF_CUDA_CHECK(ctx, cudaFuncSetAttribute(fused_obc_kernel<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fused_smem<16>(12)));
    NEGF_CUDA_CHECK(ctx, cudaFuncSetAttribute(fused_obc_kernel<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fused_smem<32>(12)));
    NEGF_CUDA_CHECK(ctx, cudaFuncSetAttribute(fused_ret_kernel<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fused_smem<16>(9)));
    NEGF_CUDA_CHECK(ctx, cudaFuncSetAttribute(fused_ret_kernel<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fused_smem<32>(9)));
    NEGF_CUDA_CHECK(ctx, cudaFuncSetAttribute(fused_lg_kernel<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fused_smem<16>(11)));
    NEGF_CUDA_CHECK(ctx, cudaFuncSetAttribute(fused_lg_kernel<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fused_smem<32>(11)));
    return NEGF_OK;
}

int fused_obc_launch(negf_ctx* ctx, const FusedObcArgs& a) {
    ProfScope _ps(ctx, NEGF_PROF_FUSED);
    const int grid = a.ns * a.ne;
    if (a.b <= 16) fused_obc_kernel<16><<<grid, FNT, fused_smem<16>(12), ctx->stream>>>(a);
    else           fused_obc_kernel<32><<<grid, FNT, fused_smem<32>(12), ctx->stream>>>(a);
    NEGF_LAUNCH_CHECK(ctx);
    return NEGF_OK;
}

int fused_ret_launch(negf_ctx* ctx, const FusedProblem& P, const FusedRetOut& o) {
    ProfScope _ps(ctx, NEGF_PROF_FUSED);
    if (P.b <= 16) fused_ret_kernel<16><<<P.ne, FNT, fused_smem<16>(9), ctx->stream>>>(P, o);
    else           fused_ret_kernel<32><<<P.ne, FNT, fused_smem<32>(9), ctx->stream>>>(P, o);
    NEGF_LAUNCH_CHECK(ctx);
    return NEGF_OK;
}

int fused_lg_launch(negf_ctx* ctx, const FusedProblem& P, const FusedLgArgs& a) {
    ProfScope _ps(ctx, NEGF_PROF_FUSED);
    const dim3 grid(P.ne, a.nx);
    if (P.b <= 16) fused_lg_kernel<16><<<grid, FNT, fused_smem<16>(11), ctx->stream>>>(P, a);
    else           fused_lg_kernel<32><<<grid, FNT, fused_smem<32>(11), ctx->stream>>>(P, a);
    NEGF_LAUNCH_CHECK(ctx);
    return NEGF_OK;
}
