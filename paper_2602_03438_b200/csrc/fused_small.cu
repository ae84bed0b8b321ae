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
//   fused_lg_kernel    S5+S6: one CTA per (energy, < or >), the hoisted forward recursion and the compact backward form
//                      as a software pipeline of two phases per step.
// Building blocks inside the CTA (all measured in-kernel with clock64, b = 16): a warp of these kernels issues about
// one instruction every three cycles (two warps per scheduler, dependent code), so every block is built for a short
// instruction path, not for pipe throughput:
//   f_phase    two to four INDEPENDENT complex products of a chain step as 8 x 8 DMMA.8x8x4 tiles spread over the
//              eight warps, one block barrier (a lone 16^3 product ~1000 cycles, four of them ~2000);
//   f_inverse  Gauss-Jordan with implicit pivoting on all eight warps (lane = row, columns cyclic over the warps),
//              ~450 cycles per column (first version, one warp: ~680);
//   staging    the next step's H blocks by cp.async.bulk (TMA, completion on an mbarrier) in the retarded sweep,
//              global -> registers -> shared memory one step ahead everywhere else.
// Same arithmetic definitions as the batched path (obc.cu, rgf.cu); results agree to rounding, not to the bit.
#include <type_traits>

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

// ---- a PHASE of independent products on the FP64 tensor pipe ---------------------------------------------------------
// The chains are sequential, but most steps hold two to four products that do not depend on each other (g u and g l;
// l g u, u g l, u g u, l g l).  A phase runs NP of them at once with ONE block barrier.  A warp here issues about one
// instruction every three cycles (two warps per scheduler, dependent code), so what a product costs is its
// instruction count: on the plain FP64 pipe a 16 x 16 x 16 complex product was ~250 instructions per thread
// (1050 cycles); as DMMA.8x8x4 it is 8 x 8 output tiles of 4 k-steps x (2 LDS.128 + 4 DMMA): the interleaved
// (re, im) element one lane loads IS its A (or B) fragment of both the real and the imaginary operand, and the four
// accumulators rr, ii, ri, ir (re = rr - ii, im = ri + ir; conjugated B: re = rr + ii, im = ir - ri) are independent
// chains.  Work units = (product, tile) spread over the eight warps; a lone 16 x 16 product splits every tile into its
// real and imaginary half (two warps per tile).  k beyond b is loaded as zero; rows / columns beyond b are not stored.
//   C = alpha * A * op(B) + beta * D + eye * I      alpha, beta real; op = identity, or conjugate transpose where bit
//   j of OPBMASK is set; a null C is an empty slot of the phase
struct Job { cplx* C; const cplx* A; const cplx* B; const cplx* D; double alpha, beta, eye; };
__device__ __forceinline__ Job job(cplx* C, const cplx* A, const cplx* B, double alpha, const cplx* D = nullptr,
                                   double beta = 0.0, double eye = 0.0) {
    Job j; j.C = C; j.A = A; j.B = B; j.D = D; j.alpha = alpha; j.beta = beta; j.eye = eye; return j;
}
__device__ __forceinline__ void dmma884(double (&c)[2], double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
                 : "+d"(c[0]), "+d"(c[1]) : "d"(a), "d"(b));
}
template <int Q, int N, class F>
__device__ __forceinline__ void f_static_for(F&& f) {
    if constexpr (Q < N) { f(std::integral_constant<int, Q>{}); f_static_for<Q + 1, N>(f); }
}
// One work unit: the 8 x 8 output tile (r0, c0) of one product; part (SPLIT only): 0 real half, 1 imaginary half.
template <int FB, bool OPB, bool SPLIT>
__device__ __forceinline__ void f_tile_mma(double (&acc)[4][2], const Job& me, int r0, int c0, int part, int b, int g, int t) {
    constexpr int LD = Mat<FB>::LD;
    const cplx* ap = me.A + (r0 + g) * LD + t;
    const cplx* bp = OPB ? me.B + (c0 + g) * LD + t : me.B + t * LD + c0 + g;
    constexpr int bstep = OPB ? 4 : 4 * LD;
    const int ksteps = (b + 3) >> 2;
#pragma unroll 2
    for (int ks = 0; ks < ksteps; ks++) {
        const bool in = 4 * ks + t < b;
        const cplx a = in ? ap[4 * ks] : cmake(0.0, 0.0);
        const cplx bv = in ? bp[ks * bstep] : cmake(0.0, 0.0);
        if (!SPLIT || part == 0) { dmma884(acc[0], a.x, bv.x); dmma884(acc[1], a.y, bv.y); }
        if (!SPLIT || part == 1) { dmma884(acc[2], a.x, bv.y); dmma884(acc[3], a.y, bv.x); }
    }
}
template <int FB, bool OPB, bool SPLIT>
__device__ __forceinline__ void f_tile_store(const double (&acc)[4][2], const Job& me, int r0, int c0, int part, int b, int g, int t) {
    constexpr int LD = Mat<FB>::LD;
    constexpr double cs = OPB ? -1.0 : 1.0;
    const int r = r0 + g;
    if (r >= b) return;
#pragma unroll
    for (int h = 0; h < 2; h++) {
        const int c = c0 + 2 * t + h;
        if (c < b) {
            double re = me.alpha * (acc[0][h] - cs * acc[1][h]);
            double im = me.alpha * (cs * acc[2][h] + acc[3][h]);
            if (me.D) { const cplx dv = me.D[r * LD + c]; re = fma(me.beta, dv.x, re); im = fma(me.beta, dv.y, im); }
            if (me.eye != 0.0 && r == c) re += me.eye;
            if (!SPLIT) me.C[r * LD + c] = cmake(re, im);
            else if (part == 0) me.C[r * LD + c].x = re;
            else me.C[r * LD + c].y = im;
        }
    }
}
// ALIAS: some C of the phase is an operand (A or B) of a product of the phase: one more barrier before the stores
// (D == C of the same product needs none: an element is read by the thread that writes it).  Ends with a barrier.
// The product a unit belongs to is resolved by a warp-uniform branch per product, so that alpha, beta, eye and a
// null D fold into the code of that branch.
template <int FB, int NP, unsigned OPBMASK = 0u, bool ALIAS = false>
__device__ __forceinline__ void f_phase(const Job (&J)[NP], int b) {
    constexpr int TD = FB / 8, T = TD * TD;                                // 8 x 8 tiles per product
    constexpr bool SPLIT = NP * T < FNT / 32;                              // real / imaginary halves on different warps
    constexpr int PARTS = SPLIT ? 2 : 1, U = NP * T * PARTS, NW = FNT / 32, UPW = (U + NW - 1) / NW;
    static_assert(NP == 1 || NP == 2 || NP == 4, "products per phase");
    static_assert(U % NW == 0 && (T * PARTS) % NW == 0 || NW % (T * PARTS) == 0, "units per warp");
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, g = lane >> 2, t = lane & 3;
    double acc[UPW][4][2];
#pragma unroll
    for (int i = 0; i < UPW; i++) {
#pragma unroll
        for (int q = 0; q < 4; q++) { acc[i][q][0] = 0.0; acc[i][q][1] = 0.0; }
        const int u = w + NW * i, jn = u / (T * PARTS), tile = (u / PARTS) % T, part = u % PARTS;
        const int r0 = (tile / TD) * 8, c0 = (tile % TD) * 8;
        if (r0 < b && c0 < b) {
            f_static_for<0, NP>([&](auto qc) {
                constexpr int q = decltype(qc)::value;
                if (jn == q && J[q].C != nullptr) f_tile_mma<FB, ((OPBMASK >> q) & 1u) != 0u, SPLIT>(acc[i], J[q], r0, c0, part, b, g, t);
            });
        }
    }
    if (ALIAS) __syncthreads();
#pragma unroll
    for (int i = 0; i < UPW; i++) {
        const int u = w + NW * i, jn = u / (T * PARTS), tile = (u / PARTS) % T, part = u % PARTS;
        const int r0 = (tile / TD) * 8, c0 = (tile % TD) * 8;
        if (r0 < b && c0 < b) {
            f_static_for<0, NP>([&](auto qc) {
                constexpr int q = decltype(qc)::value;
                if (jn == q && J[q].C != nullptr) f_tile_store<FB, ((OPBMASK >> q) & 1u) != 0u, SPLIT>(acc[i], J[q], r0, c0, part, b, g, t);
            });
        }
    }
    __syncthreads();
}

// ---- in-CTA inverse on all eight warps -------------------------------------------------------------------------------
// Gauss-Jordan with implicit threshold pivoting on the leading 32 bits of |re|+|im| (lowest row among equals).
// lane = matrix row; warp w holds the columns w, w + 8, ... in registers (2 at FB = 16, 4 at FB = 32).  Step k belongs
// to warp k % 8, whose register 0 is column k (a warp rotates its registers by one after each step it owned, so the
// step body is one piece of static code in a rolled loop).  As soon as its column is up to date the owner publishes
// it in shared memory, runs the pivot search as ONE redux on a (magnitude, row) key while EVERY lane computes the
// reciprocal of its own candidate, and the winning lane alone writes reciprocal and row index (two buffers, one block
// barrier per step); every warp then forms its rows' multipliers and updates its own columns, the pivot row's
// entries coming from lane p of the same warp by shuffle.  The next owner updates its pivot column first and
// publishes before the rest of its update.  Only the b real columns are eliminated (no padding steps).
struct FusedScratch {
    cplx col[2][32];           // pivot column of the step as it is before the step, double-buffered
    cplx dinv[2];              // 1 / pivot of the step
    double red[16];            // norm reduction
    int piv[64];               // [k] pivot row of column k; [32 + r] its inverse
    int pcur[2];               // pivot row of the step (+ 256 if the pivot was zero), double-buffered
    int sing;                  // 0 or 1-based column of the first zero pivot
    int pad;
};
constexpr int IW = FNT / 32;   // warps of the inverse
// Pivot search of one column over the lanes of a warp with ONE redux: key = the leading 27 bits of |re|+|im| (+1, so
// that an eligible zero still beats an ineligible lane) above 5 bits of 31 - lane, i.e. the largest candidate up to a
// relative 2^-15, lowest row among equals.  Exactly one lane has key == kmax (the pivot lane); kmax >> 5 <= 1: zero pivot.
__device__ __forceinline__ unsigned f_pivot_key(const cplx v, bool elig, int lane) {
    unsigned key = 0u;
    if (elig) key = ((((unsigned)((unsigned long long)__double_as_longlong(cabs1(v)) >> 32)) >> 5) + 1u) << 5 | (unsigned)(31 - lane);
    return key;
}
__device__ __forceinline__ cplx f_shfl(cplx v, int src) {
    return cmake(__shfl_sync(FULLM, v.x, src), __shfl_sync(FULLM, v.y, src));
}
// In-place inverse of the b x b block M (shared memory; `src` = where the matrix is read from, may be M).
// sh->sing = 0 or the 1-based column of the first zero pivot.  Ends with a block barrier (the caller's previous phase
// ended with one).
// A warp here issues about one instruction every three cycles (two warps per scheduler, everything dependent), so
// the time of a step is the number of instructions between the barrier and the next owner's publication: the pivot
// row is NOT scaled when it is chosen (its 1 / pivot is applied once, when the result is stored - later steps update
// an unscaled pivot row with the same formula as any other row), the winner of the redux writes the pivot itself,
// and all bookkeeping sits behind the publication in program order.
template <int FB>
__device__ __noinline__ void f_inverse(cplx* M, const cplx* src, int b, FusedScratch* sh) {
    constexpr int LD = Mat<FB>::LD, CPW = FB / IW;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const bool inb = lane < b;
    cplx x[CPW];
#pragma unroll
    for (int j = 0; j < CPW; j++) {
        const int c = w + IW * j;
        x[j] = (inb && c < b) ? src[lane * LD + c] : cmake(0.0, 0.0);
    }
    bool unused = inb;
    int pk = 0, singk = 0;
    cplx drow = cmake(1.0, 0.0);                           // 1 / pivot of the step this row was the pivot row of
    // the owner of a step publishes its column as soon as the column is up to date, then the pivot: the lane whose key
    // wins the redux writes its own reciprocal and its index (nobody else needs to learn them before the barrier)
    auto publish = [&](int buf) {
        sh->col[buf][lane] = x[0];
        const unsigned key = f_pivot_key(x[0], unused, lane);
        const unsigned kmax = __reduce_max_sync(FULLM, key);
        const cplx rc = f_recip(x[0]);
        if (key == kmax) {
            const bool zero = (kmax >> 5) <= 1u;
            sh->dinv[buf] = zero ? cmake(1.0, 0.0) : rc;
            sh->pcur[buf] = lane | (zero ? 256 : 0);
        }
        // the publisher only ARRIVES at the step's barrier (named barrier 1 + buf, all FNT threads): the other warps
        // are released now, not after the rest of the publisher's update; it reads its own publication back
        __syncwarp();
        asm volatile("bar.arrive %0, %1;" ::"r"(1 + buf), "n"(FNT) : "memory");
    };
    auto step = [&](int k, int buf) {
        if (w != (k & (IW - 1))) asm volatile("bar.sync %0, %1;" ::"r"(1 + buf), "n"(FNT) : "memory");
        const int pw = sh->pcur[buf];
        const cplx d = sh->dinv[buf];
        const cplx mr = cmul(sh->col[buf][lane], d);       // multiplier of this row
        const int pp = pw & 255;
        const bool isp = lane == pp;
        auto upd = [&](cplx t) {
            const cplx pr = f_shfl(t, pp);
            if (!isp) cfms(t, mr, pr);
            return t;
        };
        if (isp) unused = false;
        if (w == (k & (IW - 1))) {                         // owner: update and rotate, the finished column goes to the back
#pragma unroll
            for (int j = 1; j < CPW; j++) x[j - 1] = upd(x[j]);
            x[CPW - 1] = isp ? cmake(1.0, 0.0) : cneg(mr);
        } else {
            x[0] = upd(x[0]);
            if (w == ((k + 1) & (IW - 1)) && k + 1 < b) publish(buf ^ 1);      // next owner, before the rest of its update
#pragma unroll
            for (int j = 1; j < CPW; j++) x[j] = upd(x[j]);
        }
        if (isp) drow = d;
        if (lane == k) pk = pp;                            // lane k remembers the pivot row of column k
        if ((pw & 256) && !singk) singk = k + 1;
    };
    if (w == 0) publish(0);
#pragma unroll 1
    for (int k = 0; k < b; k += 2) {
        step(k, 0);
        if (k + 1 < b) step(k + 1, 1);
    }
    // lane i holds B[i][j] = X[i][piv[j]], X = Pi A^-1 (zinv.cu): A^-1[pinv[i]][piv[j]] = B[i][j]
    if (w == 0 && inb) { sh->piv[lane] = pk; sh->piv[32 + pk] = lane; }
    if (threadIdx.x == 0) sh->sing = singk;
    __syncthreads();
    const int rot = w < b ? (b - w + IW - 1) / IW : 0;    // steps this warp owned = rotations of its registers
    if (inb) {
        const int dr = sh->piv[32 + lane];
#pragma unroll
        for (int j = 0; j < CPW; j++) {
            const int c = w + IW * ((j + rot) % CPW);
            if (c < b) M[dr * LD + sh->piv[c]] = cmul(x[j], drow);
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
    { const Job J[1] = {job(tmp, A, X, -1.0, nullptr, 0.0, 1.0)}; f_phase<FB, 1>(J, b); }
    { const Job J[1] = {job(X, X, tmp, 1.0, X, 1.0)}; f_phase<FB, 1, 0u, true>(J, b); }
}

// ---- shared -> shared block copy, ends with a barrier --------------------------------------------------------------
template <int FB>
__device__ __forceinline__ void s2s(cplx* D, const cplx* S, int b) {
    constexpr int LD = Mat<FB>::LD;
    for (int idx = threadIdx.x; idx < b * b; idx += FNT) { const int o = (idx / b) * LD + idx % b; D[o] = S[o]; }
    __syncthreads();
}

// ||U||_F + ||L||_F of two blocks: one block reduction in a fixed order; result to every thread.  each(o) runs once
// per element offset o before the element is read (the caller's element-wise updates ride along).
template <int FB, class F>
__device__ __forceinline__ double f_norm_pair(const cplx* U, const cplx* L, int b, double* red, F each) {
    constexpr int LD = Mat<FB>::LD;
    double a = 0.0, c = 0.0;
    for (int idx = threadIdx.x; idx < b * b; idx += FNT) {
        const int o = (idx / b) * LD + idx % b;
        each(o);                                             // element-wise work folded into the same pass
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
__global__ void __launch_bounds__(FNT, FB <= 16 ? 2 : 1) fused_obc_kernel(const FusedObcArgs a) {
    constexpr int LD = Mat<FB>::LD, SZ = Mat<FB>::SZ;
    extern __shared__ __align__(16) unsigned char fsm[];
    cplx* m = reinterpret_cast<cplx*>(fsm);
    cplx *a_s = m, *a_b = m + SZ, *g = m + 2 * SZ, *u = m + 3 * SZ, *l = m + 4 * SZ, *un = m + 5 * SZ, *ln = m + 6 * SZ,
         *gu = m + 7 * SZ, *gl = m + 8 * SZ, *t = m + 9 * SZ, *U0 = m + 10 * SZ, *L0 = m + 11 * SZ;
    FusedScratch* sh = reinterpret_cast<FusedScratch*>(m + 12 * SZ);
    double* red = sh->red;
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
    const double ref = f_norm_pair<FB>(U0, L0, b, red, [](int) {});
    int iters = 0, done = 0, sing_code = 0;
    for (int it = 0; it < a.max_iter; it++) {
        f_inverse<FB>(g, a_b, b, sh);                               // g = a_b^-1
        if (sh->sing && !sing_code) sing_code = it + 1;
        f_refine<FB>(g, a_b, gu, b);
        { const Job J[2] = {job(gu, g, u, 1.0), job(gl, g, l, 1.0)}; f_phase<FB, 2>(J, b); }          // g u, g l
        { const Job J[4] = {job(t, l, gu, 1.0),                                                      // l g u
                            job(a_b, u, gl, -1.0, a_b, 1.0),                                         // a_b -= u g l
                            job(un, u, gu, -1.0), job(ln, l, gl, -1.0)};                             // -u g u, -l g l
          f_phase<FB, 4>(J, b); }
        cplx* sw = u; u = un; un = sw; sw = l; l = ln; ln = sw;
        iters = it + 1;
        // a_s -= l g u, a_b -= l g u and the norms of the new u, l in one pass
        const double nrm = f_norm_pair<FB>(u, l, b, red, [&](int o) { a_s[o] = csub(a_s[o], t[o]); a_b[o] = csub(a_b[o], t[o]); });
        if (nrm <= a.tol * ref) { done = 1; break; }                // reading R3 (uniform over the CTA)
    }
    s2s<FB>(g, a_s, b);
    f_inverse<FB>(a_s, a_s, b, sh);                                 // g_s = a_s^-1
    if (sh->sing && !sing_code) sing_code = a.max_iter + 1;
    f_refine<FB>(a_s, g, gu, b);
    { const Job J[1] = {job(gu, a_s, U0, 1.0)}; f_phase<FB, 1>(J, b); }
    { const Job J[1] = {job(t, L0, gu, 1.0)}; f_phase<FB, 1>(J, b); }   // Sigma^R (exchanged storage: a_u g_s a_l for a right lead)
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

// ---- bulk-copy (TMA) staging of the next step's Hamiltonian blocks --------------------------------------------------
// The blocks of H are contiguous b x b x 16 B in global memory: one `cp.async.bulk` per block (the 1D form of the TMA
// unit, SASS UBLKCP) brings the NEXT step's H_ii and H_{i-1,i} into a staging area of shared memory while the CTA
// inverts the current block; completion is an mbarrier transaction count, so no thread waits on a global load.
__device__ __forceinline__ unsigned s_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(s_u32(bar)), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(s_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, unsigned bytes, unsigned long long* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(s_u32(dst)), "l"(src), "r"(bytes), "r"(s_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
    unsigned ok;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(s_u32(bar)), "r"(parity) : "memory");
    } while (!ok);
}

// Blocks of A = z S - H - Sigma^R of sweep step i for batch entry e, from the staged H blocks: M = A_ii and, for i > 0,
// U = A_{i-1,i}, A1 = A_{i,i-1} (the dagger of the upper arrays of H and S, written transposed).  S and the dense
// Sigma^R_S families, where present, are read from global memory here.  No trailing barrier.
template <int FB>
__device__ __forceinline__ void assemble_step(cplx* M, cplx* A1, cplx* U, const FusedProblem& P, int e, int i,
                                              const cplx* st_hd, const cplx* st_hu) {
    constexpr int LD = Mat<FB>::LD;
    const int b = P.b, n = P.n;
    const size_t bb = (size_t)b * b;
    const cplx z = cmake(P.energy[e], P.eta);
    const size_t kk = P.kidx ? (size_t)P.kidx[e] : 0;
    const cplx* Sd = P.Sd ? P.Sd + (kk * n + i) * bb : nullptr;
    const cplx* Su = (P.Su && i > 0) ? P.Su + (kk * (n - 1) + i - 1) * bb : nullptr;
    const bool bt = P.sr_kind == NEGF_SIGMA_BT;
    const cplx* sgd = bt ? P.sr_diag + ((size_t)e * n + i) * bb : nullptr;
    const cplx* sgu = (bt && i > 0) ? P.sr_upper + ((size_t)e * (n - 1) + i - 1) * bb : nullptr;
    const cplx* sgl = (bt && i > 0) ? P.sr_lower + ((size_t)e * (n - 1) + i - 1) * bb : nullptr;
    const cplx* bnd = (i == 0 && P.sr_left) ? P.sr_left + (size_t)e * bb : nullptr;
    const cplx* bnd2 = (i == n - 1 && P.sr_right) ? P.sr_right + (size_t)e * bb : nullptr;
    const cplx sc = P.sr_kind == NEGF_SIGMA_SCALAR ? P.sr_scalar[e] : cmake(0.0, 0.0);
    for (int idx = threadIdx.x; idx < b * b; idx += FNT) {
        const int r = idx / b, c = idx % b;
        cplx v = Sd ? cmul(z, Sd[idx]) : (r == c ? z : cmake(0.0, 0.0));
        v = csub(v, st_hd[idx]);
        if (sgd) v = csub(v, sgd[idx]);
        if (bnd) v = csub(v, bnd[idx]);
        if (bnd2) v = csub(v, bnd2[idx]);
        if (r == c) v = csub(v, sc);
        M[r * LD + c] = v;
        if (i > 0) {
            const cplx hu = st_hu[idx];
            cplx up = cmake(0.0, 0.0), lo = cmake(0.0, 0.0);
            if (Su) { const cplx su = Su[idx]; up = cmul(z, su); lo = cmul(z, cconj(su)); }
            up = csub(up, hu); lo = csub(lo, cconj(hu));
            if (sgu) up = csub(up, sgu[idx]);
            if (sgl) lo = csub(lo, sgl[c * b + r]);
            U[r * LD + c] = up;
            A1[c * LD + r] = lo;
        }
    }
}
template <int FB>
__device__ __forceinline__ void s2g_nb(cplx* g, const cplx* S, int b) {       // shared -> global, no barrier
    constexpr int LD = Mat<FB>::LD;
    if (g) for (int idx = threadIdx.x; idx < b * b; idx += FNT) g[idx] = S[(idx / b) * LD + idx % b];
}

// ---------------------------------------------------------------------------------------------------------------------
// S1 + S3 + S4: retarded sweeps, one CTA per energy
// ---------------------------------------------------------------------------------------------------------------------
// Forward step i: {Y_{i-1} = A_{i,i-1} g_{i-1}, X_{i-1} = g_{i-1} A_{i-1,i}} as one phase, M = A_ii - Y_{i-1} A_{i-1,i},
// g_i = M^-1; H_{i+1,i+1} and H_{i,i+1} arrive by bulk copy meanwhile.  Backward step i: {G_{i,i+1} = -X_i G_{i+1,i+1},
// G_{i+1,i} = -G_{i+1,i+1} Y_i, corner column} as one phase, G_ii = g_i - G_{i,i+1} Y_i; g, X, Y of step i - 1 are
// loaded into registers before the products and parked in shared memory after them.
template <int FB>
__global__ void __launch_bounds__(FNT, FB <= 16 ? 2 : 1) fused_ret_kernel(const FusedProblem P, const FusedRetOut o) {
    constexpr int SZ = Mat<FB>::SZ, LD = Mat<FB>::LD, EPT = (FB * FB + FNT - 1) / FNT;
    extern __shared__ __align__(16) unsigned char fsm[];
    cplx* m = reinterpret_cast<cplx*>(fsm);
    cplx *M = m, *gp = m + SZ, *A1 = m + 2 * SZ, *U = m + 3 * SZ, *Y = m + 4 * SZ, *X = m + 5 * SZ, *G = m + 6 * SZ,
         *Gn = m + 7 * SZ, *col = m + 8 * SZ, *col2 = m + 9 * SZ;
    FusedScratch* sh = reinterpret_cast<FusedScratch*>(m + 10 * SZ);
    cplx* st_hd = reinterpret_cast<cplx*>(sh + 1);
    cplx* st_hu = st_hd + FB * FB;
    unsigned long long* bar = reinterpret_cast<unsigned long long*>(st_hu + FB * FB);
    const int b = P.b, n = P.n, e = blockIdx.x;
    const size_t bb = (size_t)b * b;
    const unsigned blk_bytes = (unsigned)(bb * sizeof(cplx));
    const size_t kk = P.kidx ? (size_t)P.kidx[e] : 0;
    const cplx* Hd = P.Hd + kk * n * bb;
    const cplx* Hu = P.Hu ? P.Hu + kk * (n - 1) * bb : nullptr;
    cplx* Wg = o.g + (size_t)e * n * bb;
    cplx* WX = o.X + (size_t)e * (n - 1) * bb;
    cplx* WY = o.Y + (size_t)e * (n - 1) * bb;
    int code = 0;
    if (threadIdx.x == 0) mbar_init(bar, 1);
    __syncthreads();
    if (threadIdx.x == 0) { mbar_expect_tx(bar, blk_bytes); bulk_g2s(st_hd, Hd, blk_bytes, bar); }
    unsigned parity = 0;
    // S3: g_0 = A_00^-1; Y_{i-1} = A_{i,i-1} g_{i-1}; g_i = (A_ii - Y_{i-1} A_{i-1,i})^-1
    for (int i = 0; i < n; i++) {
        mbar_wait(bar, parity); parity ^= 1u;
        assemble_step<FB>(M, A1, U, P, e, i, st_hd, st_hu);
        __syncthreads();                                                  // blocks assembled, staging area free
        if (threadIdx.x == 0 && i + 1 < n) {
            mbar_expect_tx(bar, 2 * blk_bytes);
            bulk_g2s(st_hd, Hd + (size_t)(i + 1) * bb, blk_bytes, bar);
            bulk_g2s(st_hu, Hu + (size_t)i * bb, blk_bytes, bar);
        }
        if (i > 0) {
            { const Job J[2] = {job(Y, A1, gp, 1.0), job(X, gp, U, 1.0)}; f_phase<FB, 2>(J, b); }
            s2g_nb<FB>(WY + (size_t)(i - 1) * bb, Y, b);
            s2g_nb<FB>(WX + (size_t)(i - 1) * bb, X, b);
            { const Job J[1] = {job(M, Y, U, -1.0, M, 1.0)}; f_phase<FB, 1>(J, b); }
        }
        f_inverse<FB>(M, M, b, sh);
        if (sh->sing && !code) code = i + 1;
        s2g_nb<FB>(Wg + (size_t)i * bb, M, b);
        cplx* sw = gp; gp = M; M = sw;                                    // g_{i} stays resident for the next step
    }
    // S4: G_{n-1,n-1} = g_{n-1}; G_{i,i+1} = -X_i G_{i+1,i+1}; G_{i+1,i} = -G_{i+1,i+1} Y_i;
    //     G_ii = g_i - G_{i,i+1} Y_i; corner column G_{i,n-1} = -X_i G_{i+1,n-1}
    cplx rg[EPT], rx[EPT], ry[EPT];
    auto issue = [&](int i) {
#pragma unroll
        for (int q = 0; q < EPT; q++) {
            const int idx = threadIdx.x + q * FNT;
            if (idx < b * b) { rg[q] = Wg[(size_t)i * bb + idx]; rx[q] = WX[(size_t)i * bb + idx]; ry[q] = WY[(size_t)i * bb + idx]; }
        }
    };
    if (n > 1) issue(n - 2);              // every thread reads back the elements it stored itself
    for (int idx = threadIdx.x; idx < b * b; idx += FNT) {
        const int oo = (idx / b) * LD + idx % b;
        const cplx v = gp[oo];
        G[oo] = v; col[oo] = v;
        o.GR_diag[((size_t)e * n + n - 1) * bb + idx] = v;
    }
    cplx *T = A1, *Gl = U;
    for (int i = n - 2; i >= 0; i--) {
#pragma unroll
        for (int q = 0; q < EPT; q++) {
            const int idx = threadIdx.x + q * FNT;
            if (idx < b * b) { const int oo = (idx / b) * LD + idx % b; gp[oo] = rg[q]; X[oo] = rx[q]; Y[oo] = ry[q]; }
        }
        __syncthreads();
        if (i > 0) issue(i - 1);
        { const Job J[4] = {job(T, X, G, -1.0), job(o.GR_lower ? Gl : nullptr, G, Y, -1.0),
                            job(o.GR_corner ? col2 : nullptr, X, col, -1.0), job(nullptr, X, G, -1.0)};
          f_phase<FB, 4>(J, b); }
        s2g_nb<FB>(o.GR_upper ? o.GR_upper + ((size_t)e * (n - 1) + i) * bb : nullptr, T, b);
        if (o.GR_lower) s2g_nb<FB>(o.GR_lower + ((size_t)e * (n - 1) + i) * bb, Gl, b);
        { const Job J[1] = {job(Gn, T, Y, -1.0, gp, 1.0)}; f_phase<FB, 1>(J, b); }
        s2g_nb<FB>(o.GR_diag + ((size_t)e * n + i) * bb, Gn, b);
        cplx* sw = G; G = Gn; Gn = sw; sw = col; col = col2; col2 = sw;
    }
    __syncthreads();
    if (o.GR_corner) s2g_nb<FB>(o.GR_corner + (size_t)e * bb, col, b);
    if (threadIdx.x == 0 && code && o.info[e] == 0) o.info[e] = code;
}

// ---------------------------------------------------------------------------------------------------------------------
// S5 + S6: lesser / greater sweeps, one CTA per (energy, < or >)
// ---------------------------------------------------------------------------------------------------------------------
// Both sweeps are software-pipelined so that a step of the chain is TWO phases, each shared with the preparation of
// the next step (which does not depend on the chain):
//   S5  g^x_i = W_i + Z_i g^x_{i-1} Z_i^H,  Z_i = g_i A_{i,i-1},  W_i = g_i B'_i g_i^H,
//       B'_i = B_ii - (V - V^H), V = Y_{i-1} B_{i-1,i}  (the hoisted form of rgf.cu, SURVEY 8(a) S5 regrouped):
//       iteration j: {T = Z_j g^x_{j-1} | Z_{j+1} = g_{j+1} A_{j+1,j} | P = g_{j+1} B'_{j+1}},
//                    {g^x_j = W_j + T Z_j^H | W_{j+1} = P g_{j+1}^H}
//   S6  T2_i = -g^x_i A_{i+1,i}^H + g_i B_{i,i+1};  Q_i = T2_i (G^R_{i+1,i+1})^H;  P_i = g^x_i - Q_i X_i^H;
//       G^x_{i,i+1} = Q_i - X_i G^x_{i+1,i+1};  G^x_ii = P_i + X_i (G^x_{i,i+1})^H:
//       iteration i: {G^x_{i,i+1} | P_i | T2_{i-1}},  {G^x_ii | Q_{i-1}}
// g, X, H_{i,i+1}, G^R and g^x of the next step travel global -> registers before the phases and registers -> shared
// memory after them.  Dense (block-tridiagonal) Sigma^<> blocks are read where they are used (two more products per
// step, not pipelined).
template <int FB>
__global__ void __launch_bounds__(FNT, FB <= 16 ? 2 : 1) fused_lg_kernel(const FusedProblem P, const FusedLgArgs a) {
    constexpr int SZ = Mat<FB>::SZ, LD = Mat<FB>::LD, EPT = (FB * FB + FNT - 1) / FNT;
    extern __shared__ __align__(16) unsigned char fsm[];
    cplx* m = reinterpret_cast<cplx*>(fsm);
    const int b = P.b, n = P.n, e = blockIdx.x;
    const FusedLgOne& S = a.x[blockIdx.y];
    const size_t bb = (size_t)b * b;
    const cplx* Wg = a.g + (size_t)e * n * bb;
    const cplx* WX = a.X + (size_t)e * (n - 1) * bb;
    const cplx* WY = a.Y + (size_t)e * (n - 1) * bb;
    const cplx* GRd = a.GR_diag + (size_t)e * n * bb;
    cplx* Wgx = S.gx + (size_t)e * n * bb;
    const bool bt = S.kind == NEGF_SIGMA_BT;
    const cplx z = cmake(P.energy[e], P.eta);
    const size_t kk = P.kidx ? (size_t)P.kidx[e] : 0;
    const cplx* Hu = P.Hu ? P.Hu + kk * (n - 1) * bb : nullptr;
    const cplx* Su = P.Su ? P.Su + kk * (n - 1) * bb : nullptr;
    const cplx* sgl = P.sr_kind == NEGF_SIGMA_BT ? P.sr_lower + (size_t)e * (n - 1) * bb : nullptr;
    // element idx of a b x b block (global, dense) <-> offset in a shared block
    auto soff = [&](int idx) { return (idx / b) * LD + idx % b; };
    // A_{i+1,i} = z S_{i,i+1}^H - H_{i,i+1}^H - Sigma^R_{i+1,i}, written transposed from the raw upper block hu
    auto put_lower = [&](cplx* A1, int i, const cplx (&hu)[EPT]) {
#pragma unroll
        for (int q = 0; q < EPT; q++) {
            const int idx = threadIdx.x + q * FNT;
            if (idx < b * b) {
                const int r = idx / b, c = idx % b;
                cplx lo = Su ? cmul(z, cconj(Su[(size_t)i * bb + idx])) : cmake(0.0, 0.0);
                lo = csub(lo, cconj(hu[q]));
                if (sgl) lo = csub(lo, sgl[(size_t)i * bb + c * b + r]);
                A1[c * LD + r] = lo;
            }
        }
    };
    auto put = [&](cplx* D, const cplx (&v)[EPT]) {
#pragma unroll
        for (int q = 0; q < EPT; q++) { const int idx = threadIdx.x + q * FNT; if (idx < b * b) D[soff(idx)] = v[q]; }
    };
    auto get = [&](cplx (&v)[EPT], const cplx* g) {
#pragma unroll
        for (int q = 0; q < EPT; q++) { const int idx = threadIdx.x + q * FNT; if (idx < b * b) v[q] = g[idx]; }
    };
    // B_ii of this family: scalar * I + dense diagonal block + boundary blocks
    auto put_B = [&](cplx* Bm, int i) {
        const cplx sc = S.kind == NEGF_SIGMA_SCALAR ? S.scalar[e] : cmake(0.0, 0.0);
        const cplx* sd = bt ? S.diag + ((size_t)e * n + i) * bb : nullptr;
        const cplx* bl = (i == 0 && S.left) ? S.left + (size_t)e * bb : nullptr;
        const cplx* br = (i == n - 1 && S.right) ? S.right + (size_t)e * bb : nullptr;
        for (int idx = threadIdx.x; idx < b * b; idx += FNT) {
            cplx v = (idx / b == idx % b) ? sc : cmake(0.0, 0.0);
            if (sd) v = cadd(v, sd[idx]);
            if (bl) v = cadd(v, bl[idx]);
            if (br) v = cadd(v, br[idx]);
            Bm[soff(idx)] = v;
        }
    };
    cplx r0[EPT], r1[EPT], r2[EPT], r3[EPT];
    // ---------------- S5 ----------------
    cplx *gx = m, *gxn = m + SZ, *Z = m + 2 * SZ, *Zn = m + 3 * SZ, *W = m + 4 * SZ, *Wn = m + 5 * SZ, *gin = m + 6 * SZ,
         *A1n = m + 7 * SZ, *Bmn = m + 8 * SZ, *Pn = m + 9 * SZ, *T = m + 10 * SZ, *E1 = m + 11 * SZ, *E2 = m + 12 * SZ;
    get(r0, Wg); put(gin, r0); put_B(Bmn, 0);
    __syncthreads();
    if (n > 1) { get(r0, Wg + bb); get(r1, Hu); }
    { const Job J[1] = {job(Pn, gin, Bmn, 1.0)}; f_phase<FB, 1>(J, b); }
    { const Job J[1] = {job(gx, Pn, gin, 1.0)}; f_phase<FB, 1, 1u>(J, b); }               // g^x_0 = g_0 B_00 g_0^H
    s2g_nb<FB>(Wgx, gx, b);
    for (int j = 0; j < n; j++) {
        const bool nxt = j + 1 < n;
        if (nxt) {
            put(gin, r0); put_lower(A1n, j, r1); put_B(Bmn, j + 1);
            if (bt) { get(r2, WY + (size_t)j * bb); get(r3, S.upper + ((size_t)e * (n - 1) + j) * bb); put(E1, r2); put(E2, r3); }
        }
        __syncthreads();
        if (j + 2 < n) { get(r0, Wg + (size_t)(j + 2) * bb); get(r1, Hu + (size_t)(j + 1) * bb); }
        if (nxt && bt) {                                                  // B'_{j+1} = B - (V - V^H), V = Y_j B_{j,j+1}
            { const Job J[1] = {job(Pn, E1, E2, 1.0)}; f_phase<FB, 1>(J, b); }
            for (int idx = threadIdx.x; idx < b * b; idx += FNT) {
                const int r = idx / b, c = idx % b;
                const cplx v = Pn[r * LD + c], vt = Pn[c * LD + r];
                cplx& d = Bmn[r * LD + c];
                d = cmake(d.x - (v.x - vt.x), d.y - (v.y + vt.y));
            }
            __syncthreads();
        }
        if (j == 0 && !nxt) break;
        { const Job J[4] = {job(j > 0 ? T : nullptr, Z, gx, 1.0), job(nxt ? Zn : nullptr, gin, A1n, 1.0),
                            job(nxt ? Pn : nullptr, gin, Bmn, 1.0), job(nullptr, gin, gin, 1.0)};
          f_phase<FB, 4>(J, b); }
        { const Job J[2] = {job(j > 0 ? gxn : nullptr, T, Z, 1.0, W, 1.0), job(nxt ? Wn : nullptr, Pn, gin, 1.0)};
          f_phase<FB, 2, 3u>(J, b); }
        if (j > 0) { s2g_nb<FB>(Wgx + (size_t)j * bb, gxn, b); cplx* sw = gx; gx = gxn; gxn = sw; }
        { cplx* sw = Z; Z = Zn; Zn = sw; sw = W; W = Wn; Wn = sw; }
    }
    // ---------------- S6 ----------------
    // G^x_{n-1,n-1} = g^x_{n-1}
    cplx *GXa = m + 9 * SZ, *GXb = m + 10 * SZ, *Xs = m + 2 * SZ, *GRn = m + 3 * SZ, *T2n = m + 4 * SZ, *Pm = m + 5 * SZ,
         *Qn = m + 6 * SZ;
    cplx* slotP[2] = {m + 7 * SZ, m + 8 * SZ};                           // A_{i,i-1} of the next step, then Q_{i-1}
    cplx* gxs[2];                                                        // g^x_i lives in gxs[i & 1]
    gxs[(n - 1) & 1] = gx; gxs[n & 1] = gxn;
    __syncthreads();
    for (int idx = threadIdx.x; idx < b * b; idx += FNT) {
        const cplx v = gx[soff(idx)];
        GXa[soff(idx)] = v;
        S.GX_diag[((size_t)e * n + n - 1) * bb + idx] = v;
    }
    if (n > 1) {
        // prologue: T2_{n-2}, Q_{n-2} (each thread reads back the g^x elements it stored itself)
        get(r0, Wgx + (size_t)(n - 2) * bb); get(r1, Hu + (size_t)(n - 2) * bb); get(r2, GRd + (size_t)(n - 1) * bb);
        get(r3, WX + (size_t)(n - 2) * bb);
        put(gxs[(n - 2) & 1], r0); put_lower(slotP[(n - 1) & 1], n - 2, r1); put(GRn, r2);
        if (bt) { get(r0, Wg + (size_t)(n - 2) * bb); get(r1, S.upper + ((size_t)e * (n - 1) + n - 2) * bb); put(E1, r0); put(E2, r1); }
        __syncthreads();
        { const Job J[1] = {job(T2n, gxs[(n - 2) & 1], slotP[(n - 1) & 1], -1.0)}; f_phase<FB, 1, 1u>(J, b); }
        if (bt) { const Job J[1] = {job(T2n, E1, E2, 1.0, T2n, 1.0)}; f_phase<FB, 1>(J, b); }
        if (n > 2) { get(r0, Wgx + (size_t)(n - 3) * bb); get(r1, Hu + (size_t)(n - 3) * bb); get(r2, GRd + (size_t)(n - 2) * bb); }
        { const Job J[1] = {job(slotP[(n - 1) & 1], T2n, GRn, 1.0)}; f_phase<FB, 1, 1u>(J, b); }       // Q_{n-2}
    }
    for (int i = n - 2; i >= 0; i--) {
        cplx* Qi = slotP[(i + 1) & 1];
        cplx* gxi = gxs[i & 1];
        const bool nxt = i > 0;
        // the registers hold X_i and, for the preparation of step i - 1, g^x_{i-1}, H_{i-1,i}, G^R_ii (loaded one step ago)
        put(Xs, r3);
        if (nxt) { put(gxs[(i - 1) & 1], r0); put_lower(slotP[i & 1], i - 1, r1); put(GRn, r2); }
        __syncthreads();
        if (i >= 1) get(r3, WX + (size_t)(i - 1) * bb);
        if (i >= 2) { get(r0, Wgx + (size_t)(i - 2) * bb); get(r1, Hu + (size_t)(i - 2) * bb); get(r2, GRd + (size_t)(i - 1) * bb); }
        { const Job J[4] = {job(Qn, Xs, GXa, -1.0, Qi, 1.0), job(Pm, Qi, Xs, -1.0, gxi, 1.0),
                            job(nxt ? T2n : nullptr, gxs[(i - 1) & 1], slotP[i & 1], -1.0), job(nullptr, Xs, Xs, 1.0)};
          f_phase<FB, 4, 6u>(J, b); }
        s2g_nb<FB>(S.GX_upper ? S.GX_upper + ((size_t)e * (n - 1) + i) * bb : nullptr, Qn, b);
        if (nxt && bt) {
            cplx t0[EPT], t1[EPT];
            get(t0, Wg + (size_t)(i - 1) * bb); get(t1, S.upper + ((size_t)e * (n - 1) + i - 1) * bb); put(E1, t0); put(E2, t1);
            __syncthreads();
            const Job J[1] = {job(T2n, E1, E2, 1.0, T2n, 1.0)}; f_phase<FB, 1>(J, b);
        }
        { const Job J[2] = {job(GXb, Xs, Qn, 1.0, Pm, 1.0), job(nxt ? slotP[i & 1] : nullptr, T2n, GRn, 1.0)};
          f_phase<FB, 2, 3u>(J, b); }
        s2g_nb<FB>(S.GX_diag + ((size_t)e * n + i) * bb, GXb, b);
        cplx* sw = GXa; GXa = GXb; GXb = sw;
    }
}

template <int FB> constexpr size_t fused_smem(int nmat) {
    return (size_t)nmat * Mat<FB>::SZ * sizeof(cplx) + sizeof(FusedScratch);
}

// retarded kernel: 10 blocks + scratch + staging area of two raw H blocks + the mbarrier
template <int FB> constexpr size_t fused_smem_ret() { return fused_smem<FB>(10) + 2 * (size_t)FB * FB * sizeof(cplx) + 16; }

}  // namespace

int fused_prepare(negf_ctx* ctx) {
    NEGF_CUDA_CHECK(ctx, cudaFuncSetAttribute(fused_obc_kernel<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fused_smem<16>(12)));
    NEGF_CUDA_CHECK(ctx, cudaFuncSetAttribute(fused_obc_kernel<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fused_smem<32>(12)));
    NEGF_CUDA_CHECK(ctx, cudaFuncSetAttribute(fused_ret_kernel<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fused_smem_ret<16>()));
    NEGF_CUDA_CHECK(ctx, cudaFuncSetAttribute(fused_ret_kernel<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fused_smem_ret<32>()));
    NEGF_CUDA_CHECK(ctx, cudaFuncSetAttribute(fused_lg_kernel<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fused_smem<16>(13)));
    NEGF_CUDA_CHECK(ctx, cudaFuncSetAttribute(fused_lg_kernel<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fused_smem<32>(13)));
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
    if (P.b <= 16) fused_ret_kernel<16><<<P.ne, FNT, fused_smem_ret<16>(), ctx->stream>>>(P, o);
    else           fused_ret_kernel<32><<<P.ne, FNT, fused_smem_ret<32>(), ctx->stream>>>(P, o);
    NEGF_LAUNCH_CHECK(ctx);
    return NEGF_OK;
}

int fused_lg_launch(negf_ctx* ctx, const FusedProblem& P, const FusedLgArgs& a) {
    ProfScope _ps(ctx, NEGF_PROF_FUSED);
    const dim3 grid(P.ne, a.nx);
    if (P.b <= 16) fused_lg_kernel<16><<<grid, FNT, fused_smem<16>(13), ctx->stream>>>(P, a);
    else           fused_lg_kernel<32><<<grid, FNT, fused_smem<32>(13), ctx->stream>>>(P, a);
    NEGF_LAUNCH_CHECK(ctx);
    return NEGF_OK;
}
