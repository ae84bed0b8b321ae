// K2: batched complex-FP64 GEMM on the FP64 tensor pipe (DMMA.8x8x4).
//
//   C[e] = alpha * op(A[e]) * op(B[e]) + beta * D[e],   op in {none, conjugate transpose}
//
// Every product of the RGF sweeps and of the Sancho-Rubio doubling goes through
// this kernel.  sm_100a has no tcgen05 kind for f64 (ptxas rejects .kind::f64), so the FP64
// tensor path is warp-level mma.sync.m8n8k4 with register operands; measured issue-rate peak
// 37.15 TFLOP/s (= 148 SMs x 1.965 GHz x 128 flop/clk), identical to the DFMA peak.
//
// Design:
//  * complex product by the 4M decomposition: four real DMMAs per 8x8x4 sub-product,
//    accumulators (re, im planes) in registers;
//  * operands stay interleaved (re, im) in shared memory, staged by 16-byte cp.async with an
//    XOR swizzle that makes every LDS.128 fragment read bank-conflict free for BOTH the
//    k-contiguous and the mn-contiguous tile layout, so conjugate-transposed operands
//    (g^H, A^H, X^H of SURVEY.md 8(a) S5-S6) cost nothing: the dagger is a transposed fragment
//    read plus a sign-bit flip (integer XOR, not an FP64 op);
//  * 3-stage cp.async pipeline, BK = 16; one fragment read feeds 4 DMMAs per sub-tile pair, so
//    shared-memory bandwidth stays < 20 % while the FP64 pipe is saturated;
//  * ragged m, n, k handled by zero-filled cp.async and predicated stores.
#include "common.cuh"

namespace {

constexpr int BK = 16;
// pipeline depth.  Measured on configs[1] (b = 64, 32x32 tiles) with the first kernel (122 registers, at most
// 4 CTAs/SM): 2 / 3 / 4 / 5 stages gave 8.77 / 8.68 / 8.80 / 9.47 ms per step - more stages cost CTAs per SM,
// which matters more than load latency.  With the per-CTA load state (84-88 registers) two stages of the
// 32x32 tiles let five CTAs share an SM: 6.63 -> 6.55 ms (six CTAs: 6.61).
template <int BM> struct StagesFor { static constexpr int value = 3; };
template <> struct StagesFor<32> { static constexpr int value = 2; };
// (16x16 tiles, configs[1] step: 2 / 3 / 4 stages = 5.90 / 5.82 / 5.94 ms: the default of 3 stays)

__device__ __forceinline__ void dmma(double& c0, double& c1, double a, double b) {
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
        : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}
__device__ __forceinline__ double flip(double x) {   // -x without touching the FP64 pipe
    return __hiloint2double(__double2hiint(x) ^ 0x80000000, __double2loint(x));
}
__device__ __forceinline__ void cp_async16(void* smem, const void* gmem, bool pred) {
    unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    int sz = pred ? 16 : 0;   // src-size 0 => 16 bytes of zeros
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" :: "r"(s), "l"(gmem), "r"(sz));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N> __device__ __forceinline__ void cp_async_wait() {
    asm volatile("cp.async.wait_group %0;\n" :: "n"(N));
}

// Tile loaders.  "KC" layout: rows indexed by the m (or n) coordinate, 16 k-elements contiguous,
// element (r, k) at r*16 + (k ^ 4*(r&1)).  "MC" layout: rows indexed by k, R mn-elements
// contiguous, element (k, r) at k*R + (r ^ 2*(k&3)).
template <int R, int NT>
__device__ __forceinline__ void load_tile_kc(cplx* sm, const cplx* g, int ld, int r0, int k0,
                                             int rmax, int kmax, int tid) {
    // global: row (r0 + r), cols k0..k0+15 contiguous
#pragma unroll
    for (int c = tid; c < R * BK; c += NT) {
        int r = c >> 4, kc = c & 15;
        bool ok = (r0 + r < rmax) && (k0 + kc < kmax);
        const cplx* src = ok ? g + (size_t)(r0 + r) * ld + (k0 + kc) : g;
        cp_async16(sm + r * BK + (kc ^ ((r & 1) << 2)), src, ok);
    }
}
template <int R, int NT>
__device__ __forceinline__ void load_tile_mc(cplx* sm, const cplx* g, int ld, int r0, int k0,
                                             int rmax, int kmax, int tid) {
    // global: row (k0 + k), cols r0..r0+R-1 contiguous
#pragma unroll
    for (int c = tid; c < R * BK; c += NT) {
        int k = c / R, r = c % R;
        bool ok = (r0 + r < rmax) && (k0 + k < kmax);
        const cplx* src = ok ? g + (size_t)(k0 + k) * ld + (r0 + r) : g;
        cp_async16(sm + k * R + (r ^ ((k & 3) << 1)), src, ok);
    }
}

// Per-thread state of one operand tile's loads, set up ONCE per CTA: the k-loop then only tests the k bound,
// issues the cp.async of its slots at fixed shared-memory offsets and advances one pointer.  (At K = 64 the
// tile loads' index arithmetic, redone for every k-block, was a third of the kernel's instructions.)
//   KC (rows = the m or n coordinate, 16 k contiguous): slot i is row r_0 + i NT/16, column kc = tid & 15
//   MC (rows = k, R mn-elements contiguous):            slot i is k-row k_0 + i NT/R, column r = tid % R
template <int R, int NT, bool KC>
struct TileLoader {
    static constexpr int ITER = R * BK / NT;
    static constexpr int RS = KC ? NT / BK : NT / R;     // rows between slots
    static_assert(R * BK % NT == 0 && (KC ? (NT % BK == 0 && RS % 2 == 0) : (NT % R == 0)), "tile/thread shape");
    const cplx* base;        // a valid address for the zero-filled copies
    const cplx* ptr;         // slot 0 of the next k-block
    long long slot_step;     // elements from slot i to slot i + 1
    long long kstep;         // elements from one k-block to the next
    unsigned soff;           // KC: shared-memory element offset of slot 0
    unsigned okmask;         // KC: bit i = row of slot i exists; MC: bit 0 = column exists
    int kin;                 // KC: kc; MC: k_0 (position inside the k-block)
    int rcol;                // MC: r

    __device__ __forceinline__ void init(const cplx* g, int ld, int r0, int rmax, int tid) {
        base = g;
        if (KC) {
            const int kc = tid & (BK - 1), r = tid / BK;
            kin = kc; rcol = 0;
            ptr = g + (size_t)(r0 + r) * ld + kc;
            slot_step = (long long)RS * ld; kstep = BK;
            soff = r * BK + (kc ^ ((r & 1) << 2));
            okmask = 0u;
#pragma unroll
            for (int i = 0; i < ITER; i++) okmask |= (r0 + r + i * RS < rmax ? 1u : 0u) << i;
        } else {
            const int r = tid % R, k = tid / R;
            kin = k; rcol = r;
            ptr = g + (size_t)k * ld + (r0 + r);
            slot_step = (long long)RS * ld; kstep = (long long)BK * ld;
            soff = 0u;
            okmask = r0 + r < rmax ? 1u : 0u;
        }
    }
    // loads of the k-block starting at k0 into the stage at sm; then points at the next k-block
    __device__ __forceinline__ void issue(cplx* sm, int k0, int kmax) {
        const cplx* p = ptr;
        if (KC) {
            const bool kok = k0 + kin < kmax;
#pragma unroll
            for (int i = 0; i < ITER; i++) {
                const bool ok = kok && ((okmask >> i) & 1u);
                cp_async16(sm + soff + i * RS * BK, ok ? p : base, ok);
                p += slot_step;
            }
        } else {
#pragma unroll
            for (int i = 0; i < ITER; i++) {
                const int k = kin + i * RS;
                const bool ok = okmask && (k0 + k < kmax);
                cp_async16(sm + k * R + (rcol ^ ((k & 3) << 1)), ok ? p : base, ok);
                p += slot_step;
            }
        }
        ptr += kstep;
    }
};

// n / d for n < 2^31 without a division: d = the divisor, (mul, sh) from GemmDiv::set on the host
__device__ __forceinline__ unsigned fastdiv(unsigned n, unsigned mul, unsigned sh) { return (__umulhi(n, mul) + n) >> sh; }

struct GemmDiv {
    unsigned tiles_n, tn_mul, tn_sh, batch, b_mul, b_sh;
    static void magic(unsigned d, unsigned& mul, unsigned& sh) {
        sh = 0; while ((1u << sh) < d) sh++;
        mul = (unsigned)(((unsigned long long)((1ull << sh) - d) << 32) / d + 1);
    }
    void set(unsigned tn, unsigned bt) { tiles_n = tn; batch = bt; magic(tn, tn_mul, tn_sh); magic(bt, b_mul, b_sh); }
};

template <int OPA, int OPB, int BM, int BN, int WM, int WN, int MINB>
__global__ void __launch_bounds__(WM * WN * 32, MINB) zgemm_kernel(const __grid_constant__ GemmGroup grp,
                                                                   const __grid_constant__ GemmDiv dv) {
    const GemmArgs& a = grp.g[blockIdx.z];
    constexpr int NT = WM * WN * 32;
    constexpr int STAGES = StagesFor<BM>::value;
    constexpr int MI = BM / WM / 8;     // 8x8 sub-tiles per warp along m
    constexpr int NI = BN / WN / 8;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* sA = reinterpret_cast<cplx*>(smem_raw);              // STAGES x BM x BK
    cplx* sB = sA + STAGES * BM * BK;                          // STAGES x BN x BK

    const unsigned e2 = fastdiv(blockIdx.y, dv.b_mul, dv.b_sh), e = blockIdx.y - e2 * dv.batch;
    // programmatic dependent launch (common.cuh): nothing of the previous kernel is read above this line
    pdl_wait();
    pdl_trigger();
    if (a.skip && a.skip[e]) return;
    const unsigned tm = fastdiv(blockIdx.x, dv.tn_mul, dv.tn_sh), tn = blockIdx.x - tm * dv.tiles_n;
    const int m0 = tm * BM, n0 = tn * BN;
    if (n0 >= a.n) return;                 // GemmGroup::ragged_n: this member has fewer column tiles than the grid
    const cplx* gA = a.A + (size_t)e * a.sA + (size_t)e2 * a.sA2;
    const cplx* gB = a.B + (size_t)e * a.sB + (size_t)e2 * a.sB2;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wm0 = (warp / WN) * (MI * 8), wn0 = (warp % WN) * (NI * 8);
    const int lr = lane >> 2, lk = lane & 3;

    double cre[MI][NI][2], cim[MI][NI][2];
#pragma unroll
    for (int i = 0; i < MI; i++)
#pragma unroll
        for (int j = 0; j < NI; j++) { cre[i][j][0] = cre[i][j][1] = cim[i][j][0] = cim[i][j][1] = 0.0; }

    const int KB = (a.k + BK - 1) / BK, kmax = a.k;
    TileLoader<BM, NT, OPA == 0> ldA;
    TileLoader<BN, NT, OPB != 0> ldB;
    ldA.init(gA, a.lda, m0, a.m, tid);
    ldB.init(gB, a.ldb, n0, a.n, tid);
    int st_issue = 0, kb_issue = 0;          // stage and k-block of the next loads (issued in order)
    auto issue = [&]() {
        if (kb_issue < KB) {
            ldA.issue(sA + st_issue * BM * BK, kb_issue * BK, kmax);
            ldB.issue(sB + st_issue * BN * BK, kb_issue * BK, kmax);
        }
        cp_async_commit();
        kb_issue++;
        st_issue = st_issue + 1 == STAGES ? 0 : st_issue + 1;
    };
#pragma unroll
    for (int s = 0; s < STAGES - 1; s++) issue();
    // beta D: the addend tile is read in the epilogue, after the last product - with one CTA per SM nothing overlaps
    // that read (rank-k updates of the blocked inverse: k = 32 .. 256, the tile read is as long as 1-3 k-blocks).
    // Ask L2 for this thread's 32-byte pieces of it now, behind the first operand loads.
    if (BM >= 64 && a.D) {
        const cplx* gDp = a.D + (size_t)e * a.sD + (size_t)e2 * a.sD2 + n0 + wn0 + lk * 2;
#pragma unroll
        for (int i = 0; i < MI; i++) {
            const int row = m0 + wm0 + i * 8 + lr;
            if (row < a.m) {
#pragma unroll
                for (int j = 0; j < NI; j++)
                    if (n0 + wn0 + lk * 2 + j * 8 < a.n)
                        asm volatile("prefetch.global.L2 [%0];" ::"l"(gDp + (size_t)row * a.ldc + j * 8));
            }
        }
    }

    int st = 0;
    for (int kb = 0; kb < KB; kb++) {
        cp_async_wait<STAGES - 2>();
        __syncthreads();
        issue();
        const cplx* tA = sA + st * BM * BK;
        const cplx* tB = sB + st * BN * BK;
        st = st + 1 == STAGES ? 0 : st + 1;
#pragma unroll
        for (int ks = 0; ks < BK / 4; ks++) {
            const int k = ks * 4 + lk;
            double ar[MI], ai[MI], an[MI], br[NI], bi[NI];
#pragma unroll
            for (int i = 0; i < MI; i++) {
                int m = wm0 + i * 8 + lr;
                cplx v = (OPA == 0) ? tA[m * BK + (k ^ ((m & 1) << 2))] : tA[k * BM + (m ^ ((k & 3) << 1))];
                ar[i] = v.x;
                // im += (sa ai) br ; re += (-sa sb ai) bi'   with bi' = |bi| sign-adjusted below
                ai[i] = (OPA == 0) ? v.y : flip(v.y);
                an[i] = ((OPA ^ OPB) == 0) ? flip(v.y) : v.y;
            }
#pragma unroll
            for (int j = 0; j < NI; j++) {
                int n = wn0 + j * 8 + lr;
                cplx v = (OPB == 0) ? tB[k * BN + (n ^ ((k & 3) << 1))] : tB[n * BK + (k ^ ((n & 1) << 2))];
                br[j] = v.x;
                bi[j] = v.y;   // raw; the conj sign of B is folded: re uses an (has -sa*sb), im uses sb below
            }
#pragma unroll
            for (int i = 0; i < MI; i++)
#pragma unroll
                for (int j = 0; j < NI; j++) {
                    dmma(cre[i][j][0], cre[i][j][1], ar[i], br[j]);
                    dmma(cim[i][j][0], cim[i][j][1], ai[i], br[j]);
                    dmma(cre[i][j][0], cre[i][j][1], an[i], bi[j]);
                    dmma(cim[i][j][0], cim[i][j][1], (OPB == 0) ? ar[i] : flip(ar[i]), bi[j]);
                }
        }
    }
    cp_async_wait<0>();

    // epilogue: C = alpha*acc + beta*D; a thread holds two adjacent columns of each 8x8 sub-tile
    const size_t eoff = (size_t)e * a.sC + (size_t)e2 * a.sC2;
    cplx* gC = a.C + eoff;
    const cplx* gD = a.D ? a.D + (size_t)e * a.sD + (size_t)e2 * a.sD2 : nullptr;
    const cplx al = a.alpha_vec ? cmul(a.alpha, a.alpha_vec[e]) : a.alpha, be = a.beta;
    const int col0 = n0 + wn0 + lk * 2, ncol = a.n;
#pragma unroll
    for (int i = 0; i < MI; i++) {
        const int row = m0 + wm0 + i * 8 + lr;
        if (row >= a.m) continue;
        const size_t roff = (size_t)row * a.ldc + col0;
        cplx* crow = gC + roff;
        const cplx* drow = gD ? gD + roff : nullptr;
#pragma unroll
        for (int j = 0; j < NI; j++) {
            const int col = col0 + j * 8;
            if (col >= ncol) continue;
            const bool two = col + 1 < ncol;
            cplx r0 = cmul(al, cmake(cre[i][j][0], cim[i][j][0]));
            cplx r1 = cmul(al, cmake(cre[i][j][1], cim[i][j][1]));
            if (drow) {
                cfma(r0, be, drow[j * 8]);
                if (two) cfma(r1, be, drow[j * 8 + 1]);
            }
            crow[j * 8] = r0;
            if (two) crow[j * 8 + 1] = r1;
        }
    }
}

// 3M variant for the compute-bound regime: per 8x8x4 sub-product THREE real DMMAs,
//   P1 = Ar Br,  P2 = Ai Bi,  P3 = (Ar + Ai)(Br + Bi);   Re = P1 - P2,  Im = P3 - P1 - P2,
// i.e. 25 % fewer tensor-pipe instructions than 4M for MI + NI extra DADDs per k-step.  The imaginary
// part is accurate norm-wise (|dIm| <~ eps (|Ar|+|Ai|)(|Br|+|Bi|)), far inside the 1e-10 bar.  Three
// accumulator sets cost registers, hence 32x24 warp tiles (128x48 CTA tiles, 8 warps).
template <int OPA, int OPB, int BM, int BN, int WM, int WN>
__global__ void __launch_bounds__(WM * WN * 32, 1) zgemm3m_kernel(const __grid_constant__ GemmGroup grp,
                                                                  const __grid_constant__ GemmDiv dv) {
    const GemmArgs& a = grp.g[blockIdx.z];
    constexpr int NT = WM * WN * 32;
    constexpr int STAGES = 3;
    constexpr int MI = BM / WM / 8;
    constexpr int NI = BN / WN / 8;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* sA = reinterpret_cast<cplx*>(smem_raw);
    cplx* sB = sA + STAGES * BM * BK;

    const unsigned e2 = fastdiv(blockIdx.y, dv.b_mul, dv.b_sh), e = blockIdx.y - e2 * dv.batch;
    if (a.skip && a.skip[e]) return;
    const unsigned tm = fastdiv(blockIdx.x, dv.tn_mul, dv.tn_sh), tn = blockIdx.x - tm * dv.tiles_n;
    const int m0 = tm * BM, n0 = tn * BN;
    if (n0 >= a.n) return;                 // GemmGroup::ragged_n: this member has fewer column tiles than the grid
    const cplx* gA = a.A + (size_t)e * a.sA + (size_t)e2 * a.sA2;
    const cplx* gB = a.B + (size_t)e * a.sB + (size_t)e2 * a.sB2;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wm0 = (warp / WN) * (MI * 8), wn0 = (warp % WN) * (NI * 8);
    const int lr = lane >> 2, lk = lane & 3;

    double p1[MI][NI][2], p2[MI][NI][2], p3[MI][NI][2];
#pragma unroll
    for (int i = 0; i < MI; i++)
#pragma unroll
        for (int j = 0; j < NI; j++)
#pragma unroll
            for (int q = 0; q < 2; q++) { p1[i][j][q] = 0.0; p2[i][j][q] = 0.0; p3[i][j][q] = 0.0; }

    const int KB = (a.k + BK - 1) / BK, kmax = a.k;
    // B tiles of 48 columns do not divide evenly over the threads in the mn-contiguous layout: old loaders there
    constexpr bool FAST_B = (OPB != 0) ? (NT % BK == 0 && (NT / BK) % 2 == 0 && BN * BK % NT == 0) : (NT % BN == 0 && BN * BK % NT == 0);
    TileLoader<BM, NT, OPA == 0> ldA;
    ldA.init(gA, a.lda, m0, a.m, tid);
    TileLoader<FAST_B ? BN : NT, NT, OPB != 0> ldB;
    if (FAST_B) ldB.init(gB, a.ldb, n0, a.n, tid);
    int st_issue = 0, kb_issue = 0;
    auto issue = [&]() {
        if (kb_issue < KB) {
            ldA.issue(sA + st_issue * BM * BK, kb_issue * BK, kmax);
            if (FAST_B) ldB.issue(sB + st_issue * BN * BK, kb_issue * BK, kmax);
            else if (OPB == 0) load_tile_mc<BN, NT>(sB + st_issue * BN * BK, gB, a.ldb, n0, kb_issue * BK, a.n, a.k, tid);
            else               load_tile_kc<BN, NT>(sB + st_issue * BN * BK, gB, a.ldb, n0, kb_issue * BK, a.n, a.k, tid);
        }
        cp_async_commit();
        kb_issue++;
        st_issue = st_issue + 1 == STAGES ? 0 : st_issue + 1;
    };
#pragma unroll
    for (int s = 0; s < STAGES - 1; s++) issue();

    int st = 0;
    for (int kb = 0; kb < KB; kb++) {
        cp_async_wait<STAGES - 2>();
        __syncthreads();
        issue();
        const cplx* tA = sA + st * BM * BK;
        const cplx* tB = sB + st * BN * BK;
        st = st + 1 == STAGES ? 0 : st + 1;
#pragma unroll
        for (int ks = 0; ks < BK / 4; ks++) {
            const int k = ks * 4 + lk;
            double ar[MI], ai[MI], as[MI], br[NI], bi[NI], bs[NI];
#pragma unroll
            for (int i = 0; i < MI; i++) {
                int m = wm0 + i * 8 + lr;
                cplx v = (OPA == 0) ? tA[m * BK + (k ^ ((m & 1) << 2))] : tA[k * BM + (m ^ ((k & 3) << 1))];
                ar[i] = v.x; ai[i] = (OPA == 0) ? v.y : flip(v.y); as[i] = ar[i] + ai[i];
            }
#pragma unroll
            for (int j = 0; j < NI; j++) {
                int n = wn0 + j * 8 + lr;
                cplx v = (OPB == 0) ? tB[k * BN + (n ^ ((k & 3) << 1))] : tB[n * BK + (k ^ ((n & 1) << 2))];
                br[j] = v.x; bi[j] = (OPB == 0) ? v.y : flip(v.y); bs[j] = br[j] + bi[j];
            }
#pragma unroll
            for (int i = 0; i < MI; i++)
#pragma unroll
                for (int j = 0; j < NI; j++) {
                    dmma(p1[i][j][0], p1[i][j][1], ar[i], br[j]);
                    dmma(p2[i][j][0], p2[i][j][1], ai[i], bi[j]);
                    dmma(p3[i][j][0], p3[i][j][1], as[i], bs[j]);
                }
        }
    }
    cp_async_wait<0>();

    cplx* gC = a.C + (size_t)e * a.sC + (size_t)e2 * a.sC2;
    const cplx* gD = a.D ? a.D + (size_t)e * a.sD + (size_t)e2 * a.sD2 : nullptr;
    const cplx al = a.alpha_vec ? cmul(a.alpha, a.alpha_vec[e]) : a.alpha, be = a.beta;
    const int col0 = n0 + wn0 + lk * 2, ncol = a.n;
#pragma unroll
    for (int i = 0; i < MI; i++) {
        const int row = m0 + wm0 + i * 8 + lr;
        if (row >= a.m) continue;
        const size_t roff = (size_t)row * a.ldc + col0;
        cplx* crow = gC + roff;
        const cplx* drow = gD ? gD + roff : nullptr;
#pragma unroll
        for (int j = 0; j < NI; j++) {
            const int col = col0 + j * 8;
            if (col >= ncol) continue;
            const bool two = col + 1 < ncol;
            cplx r0 = cmul(al, cmake(p1[i][j][0] - p2[i][j][0], (p3[i][j][0] - p1[i][j][0]) - p2[i][j][0]));
            cplx r1 = cmul(al, cmake(p1[i][j][1] - p2[i][j][1], (p3[i][j][1] - p1[i][j][1]) - p2[i][j][1]));
            if (drow) {
                cfma(r0, be, drow[j * 8]);
                if (two) cfma(r1, be, drow[j * 8 + 1]);
            }
            crow[j * 8] = r0;
            if (two) crow[j * 8 + 1] = r1;
        }
    }
}

constexpr int M3_BN = 48;      // 32x24 warp tiles: the widest that keep three accumulator sets in registers

template <int OPA, int OPB>
int launch_3m(negf_ctx* ctx, const GemmGroup& grp) {
    constexpr int BM = 128, BN = M3_BN, WM = 4, WN = 2;
    const GemmArgs& a = grp.g[0];
    constexpr int smem = 3 * (BM + BN) * BK * (int)sizeof(cplx);
    const int tiles_n = (a.n + BN - 1) / BN;
    int tiles = ((a.m + BM - 1) / BM) * tiles_n;
    dim3 grid(tiles, a.batch * a.batch2, grp.ng);
    GemmDiv dv;
    dv.set((unsigned)tiles_n, (unsigned)a.batch);
    zgemm3m_kernel<OPA, OPB, BM, BN, WM, WN><<<grid, WM * WN * 32, smem, ctx->stream>>>(grp, dv);
    NEGF_LAUNCH_CHECK(ctx);
    return NEGF_OK;
}

template <int OPA, int OPB, int BM, int BN, int WM, int WN, int MINB>
int launch_cfg(negf_ctx* ctx, const GemmGroup& grp) {
    const GemmArgs& a = grp.g[0];
    auto kern = zgemm_kernel<OPA, OPB, BM, BN, WM, WN, MINB>;
    constexpr int smem = StagesFor<BM>::value * (BM + BN) * BK * (int)sizeof(cplx);
    const int tiles_n = (a.n + BN - 1) / BN;
    int tiles = ((a.m + BM - 1) / BM) * tiles_n;
    dim3 grid(tiles, a.batch * a.batch2, grp.ng);
    GemmDiv dv;
    dv.set((unsigned)tiles_n, (unsigned)a.batch);
    // the small tiles are the latency-bound chain steps: programmatic dependent launch (common.cuh)
    if (BM <= 32) NEGF_CUDA_CHECK(ctx, launch_chain(ctx, kern, grid, dim3(WM * WN * 32), (size_t)smem, grp, dv));
    else kern<<<grid, WM * WN * 32, smem, ctx->stream>>>(grp, dv);
    NEGF_LAUNCH_CHECK(ctx);
    return NEGF_OK;
}

template <int BM, int BN, int WM, int WN, int MINB>
int launch_ops(negf_ctx* ctx, const GemmGroup& grp) {
    const GemmArgs& a = grp.g[0];
    if (a.opA == 0 && a.opB == 0) return launch_cfg<0, 0, BM, BN, WM, WN, MINB>(ctx, grp);
    if (a.opA == 1 && a.opB == 0) return launch_cfg<1, 0, BM, BN, WM, WN, MINB>(ctx, grp);
    if (a.opA == 0 && a.opB == 1) return launch_cfg<0, 1, BM, BN, WM, WN, MINB>(ctx, grp);
    return launch_cfg<1, 1, BM, BN, WM, WN, MINB>(ctx, grp);
}

}  // namespace

namespace {
template <int BM, int BN, int WM, int WN, int MINB>
cudaError_t prepare_cfg() {
    constexpr int smem = StagesFor<BM>::value * (BM + BN) * BK * (int)sizeof(cplx);
    cudaError_t e = cudaFuncSetAttribute(zgemm_kernel<0, 0, BM, BN, WM, WN, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(zgemm_kernel<1, 0, BM, BN, WM, WN, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(zgemm_kernel<0, 1, BM, BN, WM, WN, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(zgemm_kernel<1, 1, BM, BN, WM, WN, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    return e;
}
}  // namespace

// dynamic shared-memory limits of every instantiation, once per context (never inside a stream capture)
int zgemm_prepare(negf_ctx* ctx) {
    NEGF_CUDA_CHECK(ctx, (prepare_cfg<128, 64, 4, 2, 1>()));
    NEGF_CUDA_CHECK(ctx, (prepare_cfg<64, 64, 2, 2, 2>()));
    NEGF_CUDA_CHECK(ctx, (prepare_cfg<64, 64, 2, 4, 2>()));
    NEGF_CUDA_CHECK(ctx, (prepare_cfg<32, 32, 2, 2, 5>()));
    NEGF_CUDA_CHECK(ctx, (prepare_cfg<16, 16, 2, 2, 6>()));
    {
        constexpr int smem = 3 * (128 + M3_BN) * BK * (int)sizeof(cplx);
        NEGF_CUDA_CHECK(ctx, cudaFuncSetAttribute(zgemm3m_kernel<0, 0, 128, M3_BN, 4, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        NEGF_CUDA_CHECK(ctx, cudaFuncSetAttribute(zgemm3m_kernel<1, 0, 128, M3_BN, 4, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        NEGF_CUDA_CHECK(ctx, cudaFuncSetAttribute(zgemm3m_kernel<0, 1, 128, M3_BN, 4, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        NEGF_CUDA_CHECK(ctx, cudaFuncSetAttribute(zgemm3m_kernel<1, 1, 128, M3_BN, 4, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    }
    return NEGF_OK;
}

int zgemm_launch_group(negf_ctx* ctx, const GemmGroup& grp) {
    ProfScope _ps(ctx, NEGF_PROF_GEMM);
    if (grp.ng < 1 || grp.ng > NEGF_GEMM_GROUP_MAX) return NEGF_EINVAL;
    if (grp.ragged_n) {                     // lay the grid out for the widest member: it goes first
        int w = 0;
        for (int i = 1; i < grp.ng; i++) if (grp.g[i].n > grp.g[w].n) w = i;
        if (grp.g[w].n <= 0) return NEGF_OK;
        if (w != 0) { GemmGroup h = grp; h.g[0] = grp.g[w]; h.g[w] = grp.g[0]; return zgemm_launch_group(ctx, h); }
    }
    const GemmArgs& a = grp.g[0];
    if (a.m <= 0 || a.n <= 0 || a.batch <= 0) return NEGF_OK;
    if (a.k < 0 || (a.opA | a.opB) & ~1) return NEGF_EINVAL;
    if (a.batch2 < 1 || (long long)a.batch * a.batch2 > 65535) return NEGF_EUNSUPPORTED;
    for (int i = 1; i < grp.ng; i++) {      // one grid serves every member: same shape, ops and batch
        const GemmArgs& o = grp.g[i];
        if (o.m != a.m || (o.n != a.n && !grp.ragged_n) || o.k != a.k || o.opA != a.opA || o.opB != a.opB ||
            o.batch != a.batch || o.batch2 != a.batch2)
            return NEGF_EINVAL;
    }
    // In-place products.  C == A is safe only when one CTA owns all n columns of the rows it reads (every read of
    // a CTA is complete before its first store: the last k-block's wait + barrier precede the epilogue), so the
    // caller flags it and gets a tile with BN >= n; unflagged aliasing of C with an operand is rejected when
    // more than one CTA would share the operand's rows / columns.
    bool alias_a = false;
    for (int i = 0; i < grp.ng; i++) {
        const GemmArgs& o = grp.g[i];
        if (o.c_aliases_a) { alias_a = true; if (o.n > 64 || o.opA != 0) return NEGF_EINVAL; continue; }
        if ((const cplx*)o.C == o.A && o.n > 16) return NEGF_EINVAL;
        if ((const cplx*)o.C == o.B && o.m > 16) return NEGF_EINVAL;
    }
    // Tile choice: the largest CTA tile that still gives every SM work.  128x64 (8 warps, 32x32 warp
    // tiles, 1 CTA/SM) in the compute-bound regime; 64x64 (4 warps); 32x32 (4 warps of 16x16, up to
    // 4 CTAs/SM) when the batch of small blocks would otherwise leave most SMs idle.
    const long long per = (long long)a.batch * a.batch2 * grp.ng;
    const long long t128 = (long long)((a.m + 127) / 128) * ((a.n + 63) / 64) * per;
    const long long t64 = (long long)((a.m + 63) / 64) * ((a.n + 63) / 64) * per;
    if (ctx->gemm_3m && a.m > 64 && t128 >= ctx->num_sms) {     // opt-in, compute-bound regime only
        if (a.opA == 0 && a.opB == 0) return launch_3m<0, 0>(ctx, grp);
        if (a.opA == 1 && a.opB == 0) return launch_3m<1, 0>(ctx, grp);
        if (a.opA == 0 && a.opB == 1) return launch_3m<0, 1>(ctx, grp);
        return launch_3m<1, 1>(ctx, grp);
    }
    // Compute-bound regime: 64x64 tiles, TWO CTAs per SM.  The 128x64 tile (8 warps, 243 registers) leaves one
    // CTA per SM, so nothing runs while it fills its pipeline, waits at its k-block barriers, reads the addend and stores
    // its tile; two co-resident CTAs cover each other (numbers below: 4 warps of 32x32 per CTA).  Measured (kernel_bench, fraction of the FP64 peak, 128x64 -> 64x64
    // x 2): b = 2048 batch 8: 92.4 -> 94.8 %; b = 1024 batch 32: 91.5 -> 94.3 %; b = 512 batch 32: 88.6 -> 91.7 %; b = 256
    // batch 512: 86.3 -> 91.0 %; b = 300 batch 40: 51.6 -> 64.7 %; blocked inverse b = 2048 batch 8: 26.4 -> 25.6 ms;
    // whole path configs[2] 1799 -> 1723 ms, configs[3] 13.37 -> 13.00 s, configs[4] 13.13 -> 12.77 s.
    // 8 warps of 32x16 per CTA (128 registers) measured another 0.3-0.7 points above 4 warps of 32x32 (230 registers).
    if (a.m > 64 && t64 >= 2LL * ctx->num_sms && !alias_a) return launch_ops<64, 64, 2, 4, 2>(ctx, grp);
    if (a.m > 64 && t128 >= ctx->num_sms) return launch_ops<128, 64, 4, 2, 1>(ctx, grp);
    // blocks up to 64 x 64: four 32x32 CTAs per product balance the SMs better than one 64x64 CTA
    // (measured 5-7 % faster at b = 64 for 128 .. 512 products per launch)
    if ((a.m > 64 || a.n > 64) && t64 >= ctx->num_sms) return launch_ops<64, 64, 2, 2, 2>(ctx, grp);
    // launches of fewer than two 32x32 tiles per SM (the sequential chain steps: one b = 64 product per energy) are
    // bound by the length of one warp's DMMA chain, not by the pipe: 16x16 tiles (4 warps of 8x8) quarter that chain.
    // Measured on configs[1] with the threshold at 1 / 2 / 4 / always: 2 is best (5.97 -> 5.83 ms per step as 4
    // energy groups, 6.41 -> 6.11 ms on one stream; always: 6.00 / 6.26 ms).
    if (alias_a && a.n > 32) return launch_ops<64, 64, 2, 2, 2>(ctx, grp);
    const long long t32 = (long long)((a.m + 31) / 32) * ((a.n + 31) / 32) * per;
    if (t32 < 2LL * ctx->num_sms && !(alias_a && a.n > 16)) return launch_ops<16, 16, 2, 2, 6>(ctx, grp);
    return launch_ops<32, 32, 2, 2, 5>(ctx, grp);
}

int zgemm_launch(negf_ctx* ctx, const GemmArgs& a) {
    GemmGroup grp;
    grp.g[0] = a; grp.ng = 1;
    return zgemm_launch_group(ctx, grp);
}

GemmArgs zgemm_bb_args(int opA, int opB, int b, cplx alpha, const cplx* A, long long sA, const cplx* B, long long sB,
                       cplx beta, const cplx* D, long long sD, cplx* C, long long sC, int batch, const int* skip) {
    GemmArgs g;
    g.opA = opA; g.opB = opB; g.m = g.n = g.k = b; g.alpha = alpha; g.beta = beta;
    g.A = A; g.lda = b; g.sA = sA; g.B = B; g.ldb = b; g.sB = sB;
    g.D = D; g.sD = sD; g.C = C; g.ldc = b; g.sC = sC; g.batch = batch; g.skip = skip;
    g.batch2 = 1; g.sA2 = g.sB2 = g.sD2 = g.sC2 = 0; g.alpha_vec = nullptr;
    return g;
}
int zgemm_bb(negf_ctx* ctx, int opA, int opB, int b, cplx alpha, const cplx* A, long long sA,
             const cplx* B, long long sB, cplx beta, const cplx* D, long long sD,
             cplx* C, long long sC, int batch, const int* skip) {
    return zgemm_launch(ctx, zgemm_bb_args(opA, opB, b, alpha, A, sA, B, sB, beta, D, sD, C, sC, batch, skip));
}

extern "C" int negf_zgemm_batched(negf_ctx* ctx, int opA, int opB, int m, int n, int k,
                                  negf_c128 alpha, const negf_c128* A, int lda, long long strideA,
                                  const negf_c128* B, int ldb, long long strideB,
                                  negf_c128 beta, const negf_c128* D,
                                  negf_c128* C, int ldc, long long strideC, int batch) {
    if (!ctx || !A || !B || !C || m < 0 || n < 0 || k < 0 || batch < 0) return NEGF_EINVAL;
    GemmArgs g;
    g.opA = opA; g.opB = opB; g.m = m; g.n = n; g.k = k;
    g.alpha = cmake(alpha.re, alpha.im); g.beta = cmake(beta.re, beta.im);
    g.A = (const cplx*)A; g.lda = lda; g.sA = strideA;
    g.B = (const cplx*)B; g.ldb = ldb; g.sB = strideB;
    g.D = (const cplx*)D; g.sD = strideC;
    g.C = (cplx*)C; g.ldc = ldc; g.sC = strideC; g.batch = batch; g.skip = nullptr;
    g.batch2 = 1; g.sA2 = g.sB2 = g.sD2 = g.sC2 = 0; g.alpha_vec = nullptr;
    return zgemm_launch(ctx, g);
}
