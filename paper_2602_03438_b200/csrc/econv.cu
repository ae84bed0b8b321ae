// Eq. 3 of the paper: energy convolution B(E) ~ int dE' (M1 C1(E - E') M2) (.) C2(E'),
// here for M1 = M2 = I and (.) = element-wise product on the selected blocks, "performed more efficiently
// in the time domain after a fast Fourier transform".  SURVEY.md 8(f) item 3: the step on the
// other side of the LSE in Fig. 1, with the (E; i,j) -> (i,j; E) transposition that the paper does with an
// all-to-all done on the fly in shared memory.
//
//   convolution  Y[m] = scale * sum_k X1[m - k] (.) op(X2[k]),          m = 0 .. 2 N_E - 2
//   correlation  Y[m] = scale * sum_k X1[k] (.) op(X2[k - (m - (N_E-1))])   (lag m - (N_E-1); = convolution with
//                the second operand reversed in energy)
// on a uniform grid of N_E energies, zero outside the grid; op = identity or complex conjugate, optionally
// with the b x b blocks of X2 transposed (the (j,i) element, as in P^<_ij(w) ~ G^<_ij(E) G^>_ji(E - w)).
//
// One CTA takes TE consecutive elements for ALL energies, as a tile s[energy][element] in shared memory (this
// IS the transposition: the FFT runs along the energy axis with the element index across threads), zero-padded
// to L = 2^p >= 2 N_E - 1.  Radix-2 decimation-in-frequency forward transforms of both operands (bit-reversed
// output), pointwise product, decimation-in-time inverse transform (natural output).  The log2 L stages run in
// passes of up to three stages on 8 points held in registers, so the tile crosses shared memory once per pass,
// not once per stage; the first forward pass reads its points straight from global memory (rows of TE
// consecutive elements), the last one multiplies, the last inverse pass writes the scaled rows to global memory.
// 2 N_E + (2 N_E - 1) complex numbers per element of HBM traffic, each touched once.
#include "common.cuh"

namespace {

constexpr int ECONV_MAXLOG = 11;          // L <= 2048, i.e. N_E <= 1024
constexpr int ECONV_LOGTILE = 10;         // 1024 points per operand and CTA (16 KB) for L <= 256

struct EconvArgs {
    int ne; long long M;
    int mode, conj2, bt;                   // bt = block size for transposing X2's blocks, 0 = none
    const cplx* X1; const cplx* X2; cplx* Y; cplx scale;
};

// The log2 L stages are split as evenly as possible into passes of at most three stages.
__host__ __device__ constexpr int econv_npass(int logl) { return (logl + 2) / 3; }
__host__ __device__ constexpr int econv_q(int logl, int ps) {
    int np = econv_npass(logl), rem = logl, q = 0;
    for (int i = 0; i <= ps; i++) { q = (rem + (np - i) - 1) / (np - i); rem -= q; }
    return q;
}
__host__ __device__ constexpr int econv_done(int logl, int ps) {      // stages done before pass ps
    int d = 0;
    for (int i = 0; i < ps; i++) d += econv_q(logl, i);
    return d;
}

// Q radix-2 decimation-in-frequency stages on 2^Q points of both operands held in registers; the points are
// SUB rows apart inside a sub-transform of size n = SUB << Q at position j (< SUB); SH = log2(L / n).  Stage
// s pairs (p, p + n/2^(s+1)): x_p = u + v, x_{p+h} = (u - v) w_{n_s}^{j_s} with n_s = n >> s, j_s = j + i SUB.
template <int Q, int SUB, int SH>
__device__ __forceinline__ void dif_regs(cplx (&x)[1 << Q], cplx (&y)[1 << Q], const cplx* tw, int j) {
    constexpr int R = 1 << Q;
#pragma unroll
    for (int s = 0; s < Q; s++) {
        const int half = R >> (s + 1);
#pragma unroll
        for (int i = 0; i < half; i++) {
            const cplx w = tw[(j + i * SUB) << (SH + s)];
#pragma unroll
            for (int g = 0; g < R; g += 2 * half) {
                cplx u = x[g + i], v = x[g + i + half];
                x[g + i] = cadd(u, v); x[g + i + half] = cmul(csub(u, v), w);
                u = y[g + i]; v = y[g + i + half];
                y[g + i] = cadd(u, v); y[g + i + half] = cmul(csub(u, v), w);
            }
        }
    }
}

// Q decimation-in-time stages of the inverse transform, points H0 rows apart, first stage half-size H0,
// position j (< H0); SH = logL - 1 - log2 H0.  Stage s pairs (m, m + 2^s): x = u +- v conj(w)^{j_s}.
template <int Q, int H0, int SH>
__device__ __forceinline__ void dit_regs(cplx (&x)[1 << Q], const cplx* tw, int j) {
    constexpr int R = 1 << Q;
#pragma unroll
    for (int s = 0; s < Q; s++) {
#pragma unroll
        for (int m = 0; m < R; m++) {
            if (m & (1 << s)) continue;
            const cplx w = cconj(tw[(j + (m & ((1 << s) - 1)) * H0) << (SH - s)]);
            const cplx u = x[m], v = cmul(x[m + (1 << s)], w);
            x[m] = cadd(u, v); x[m + (1 << s)] = csub(u, v);
        }
    }
}

// element index of the second operand: (blk, i, j) -> (blk, j, i) inside b x b blocks when asked for
__device__ __forceinline__ long long econv_el2(const EconvArgs& a, long long el) {
    if (!a.bt || el >= a.M) return el;
    if (a.M < 2147483647LL) {                               // 32-bit index arithmetic whenever it fits
        const unsigned bt = (unsigned)a.bt, bb = bt * bt, eu = (unsigned)el, blk = eu / bb, r = eu % bb;
        return (long long)(blk * bb + (r % bt) * bt + r / bt);
    }
    const long long bb = (long long)a.bt * a.bt, blk = el / bb, r = el % bb;
    return blk * bb + (r % a.bt) * a.bt + r / a.bt;
}

template <int LOGL> struct EconvShape {
    static constexpr int L = 1 << LOGL;
    // log2 of the elements per CTA: 1024-point tiles up to L = 256; beyond, at least 4 (L = 2048: 2) elements so
    // that a row of the tile is still a 64-byte (32-byte) piece of a global-memory line
    static constexpr int LT = LOGL <= 8 ? ECONV_LOGTILE - LOGL : (LOGL <= 10 ? 2 : 1);
    static constexpr int TE = 1 << LT;
    static constexpr int NP = econv_npass(LOGL);
    static constexpr int NT = (L * TE) / 8;                  // one 8-point item per thread in a 3-stage pass
    static constexpr size_t SMEM = ((size_t)2 * L * TE + L / 2) * sizeof(cplx);   // L >= 512: 64 - 144 KB
};

// Forward pass PS over the tile: its Q stages of the sub-transforms of size 2^LN, both operands.  The first
// pass takes its points straight from global memory (zero-padded; the second operand reversed in energy for
// a correlation, conjugated and block-transposed on request); the last one leaves the pointwise product in sa.
// Every row offset is a compile-time constant, so the shared-memory accesses carry immediate offsets.
template <int LOGL, int PS>
__device__ __forceinline__ void fwd_pass(const EconvArgs& a, cplx* sa, cplx* sb, const cplx* tw, long long e0) {
    using SH = EconvShape<LOGL>;
    constexpr int Q = econv_q(LOGL, PS), R = 1 << Q, LN = LOGL - econv_done(LOGL, PS), LSUB = LN - Q, SUB = 1 << LSUB;
    constexpr bool first = PS == 0, last = PS == SH::NP - 1;
    constexpr int items = (SH::L >> Q) << SH::LT;
#pragma unroll 1
    for (int idx = threadIdx.x; idx < items; idx += SH::NT) {
        const int bf = idx >> SH::LT, t = idx & (SH::TE - 1);
        const int j = bf & (SUB - 1), base = ((bf >> LSUB) << LN) + j;
        cplx* pa = sa + (base << SH::LT) + t;
        cplx* pb = sb + (base << SH::LT) + t;
        cplx x[R], y[R];
        if (first) {
            const long long el = e0 + t, el2 = econv_el2(a, el);
#pragma unroll
            for (int m = 0; m < R; m++) {
                const int k = base + m * SUB;
                x[m] = cmake(0.0, 0.0); y[m] = x[m];
                if (k < a.ne && el < a.M) {
                    x[m] = a.X1[(size_t)k * a.M + el];
                    y[m] = a.X2[(size_t)(a.mode ? a.ne - 1 - k : k) * a.M + el2];
                    if (a.conj2) y[m].y = -y[m].y;
                }
            }
        } else {
#pragma unroll
            for (int m = 0; m < R; m++) { x[m] = pa[(m * SUB) << SH::LT]; y[m] = pb[(m * SUB) << SH::LT]; }
        }
        dif_regs<Q, SUB, LOGL - LN>(x, y, tw, j);
        if (last) {
#pragma unroll
            for (int m = 0; m < R; m++) pa[(m * SUB) << SH::LT] = cmul(x[m], y[m]);
        } else {
#pragma unroll
            for (int m = 0; m < R; m++) { pa[(m * SUB) << SH::LT] = x[m]; pb[(m * SUB) << SH::LT] = y[m]; }
        }
    }
}

// Inverse pass: the stages of forward pass PS undone in reverse order (half-sizes 2^LH ...); PS == 0 is the
// last one and writes the scaled rows 0 .. 2 N_E - 2 to global memory.
template <int LOGL, int PS>
__device__ __forceinline__ void inv_pass(const EconvArgs& a, cplx* sa, const cplx* tw, long long e0, cplx sc) {
    using SH = EconvShape<LOGL>;
    constexpr int Q = econv_q(LOGL, PS), R = 1 << Q, LH = LOGL - econv_done(LOGL, PS) - Q, H0 = 1 << LH;
    constexpr bool last = PS == 0;
    constexpr int items = (SH::L >> Q) << SH::LT;
#pragma unroll 1
    for (int idx = threadIdx.x; idx < items; idx += SH::NT) {
        const int bf = idx >> SH::LT, t = idx & (SH::TE - 1);
        const int j = bf & (H0 - 1), base = ((bf >> LH) << (LH + Q)) + j;
        cplx* pa = sa + (base << SH::LT) + t;
        cplx x[R];
#pragma unroll
        for (int m = 0; m < R; m++) x[m] = pa[(m * H0) << SH::LT];
        dit_regs<Q, H0, LOGL - 1 - LH>(x, tw, j);
        if (last) {
            const long long el = e0 + t;
#pragma unroll
            for (int m = 0; m < R; m++) {
                const int row = base + m * H0;
                if (row < 2 * a.ne - 1 && el < a.M) a.Y[(size_t)row * a.M + el] = cmul(x[m], sc);
            }
        } else {
#pragma unroll
            for (int m = 0; m < R; m++) pa[(m * H0) << SH::LT] = x[m];
        }
    }
}

template <int LOGL>
__global__ void __launch_bounds__(EconvShape<LOGL>::NT) econv_kernel(EconvArgs a) {
    using SH = EconvShape<LOGL>;
    constexpr int L = SH::L, NP = SH::NP;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* sa = reinterpret_cast<cplx*>(smem_raw);          // [L][TE]
    cplx* sb = sa + L * SH::TE;                             // [L][TE]
    cplx* tw = sb + L * SH::TE;                             // [L/2]  exp(-2 pi i j / L)
    const long long e0 = (long long)blockIdx.x * SH::TE;
    for (int j = threadIdx.x; j < L / 2; j += SH::NT) {
        double sn, cs;
        sincospi(-2.0 * (double)j / (double)L, &sn, &cs);
        tw[j] = cmake(cs, sn);
    }
    __syncthreads();
    // forward transforms of both operands (decimation in frequency, bit-reversed output) and their product
    fwd_pass<LOGL, 0>(a, sa, sb, tw, e0); __syncthreads();
    if constexpr (NP > 1) { fwd_pass<LOGL, 1>(a, sa, sb, tw, e0); __syncthreads(); }
    if constexpr (NP > 2) { fwd_pass<LOGL, 2>(a, sa, sb, tw, e0); __syncthreads(); }
    if constexpr (NP > 3) { fwd_pass<LOGL, 3>(a, sa, sb, tw, e0); __syncthreads(); }
    // inverse transform (decimation in time on the bit-reversed product, natural output)
    const cplx sc = cmake(a.scale.x / L, a.scale.y / L);
    if constexpr (NP > 3) { inv_pass<LOGL, 3>(a, sa, tw, e0, sc); __syncthreads(); }
    if constexpr (NP > 2) { inv_pass<LOGL, 2>(a, sa, tw, e0, sc); __syncthreads(); }
    if constexpr (NP > 1) { inv_pass<LOGL, 1>(a, sa, tw, e0, sc); __syncthreads(); }
    inv_pass<LOGL, 0>(a, sa, tw, e0, sc);
}

template <int LOGL>
void econv_launch(const EconvArgs& a, cudaStream_t st) {
    using SH = EconvShape<LOGL>;
    const long long ctas = (a.M + SH::TE - 1) / SH::TE;
    econv_kernel<LOGL><<<(unsigned)ctas, SH::NT, SH::SMEM, st>>>(a);
}

template <int LOGL>
cudaError_t econv_optin() {
    return cudaFuncSetAttribute(econv_kernel<LOGL>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)EconvShape<LOGL>::SMEM);
}

}  // namespace

// shared-memory opt-in of the large transforms, once per context (= per device) at negf_create
int econv_prepare(negf_ctx* ctx) {
    NEGF_CUDA_CHECK(ctx, econv_optin<9>());
    NEGF_CUDA_CHECK(ctx, econv_optin<10>());
    NEGF_CUDA_CHECK(ctx, econv_optin<11>());
    return NEGF_OK;
}

extern "C" int negf_energy_convolve(negf_ctx* ctx, int n_energy, long long elems_per_energy, int transpose_block,
                                    const negf_c128* X1, const negf_c128* X2, int mode, int conj2, negf_c128 scale,
                                    negf_c128* Y) {
    if (!ctx || !X1 || !X2 || !Y || n_energy < 1 || elems_per_energy < 1 || (mode & ~1) || (conj2 & ~1)) return NEGF_EINVAL;
    if (transpose_block < 0 || (transpose_block > 0 && elems_per_energy % ((long long)transpose_block * transpose_block)))
        return NEGF_EINVAL;
    int L = 2, logL = 1;
    while (L < 2 * n_energy - 1) { L <<= 1; logL++; }
    if (logL > ECONV_MAXLOG) return NEGF_EUNSUPPORTED;     // N_E <= 1024
    EconvArgs a;
    a.ne = n_energy; a.M = elems_per_energy; a.mode = mode; a.conj2 = conj2; a.bt = transpose_block;
    a.X1 = (const cplx*)X1; a.X2 = (const cplx*)X2; a.Y = (cplx*)Y; a.scale = cmake(scale.re, scale.im);
    const int lt = logL <= 8 ? ECONV_LOGTILE - logL : (logL <= 10 ? 2 : 1);     // = EconvShape<logL>::LT
    if (((elems_per_energy + (1LL << lt) - 1) >> lt) > 2147483647LL) return NEGF_EUNSUPPORTED;
    ProfScope _ps(ctx, NEGF_PROF_ELEMENTWISE);
    switch (logL) {
        case 1: econv_launch<1>(a, ctx->stream); break;
        case 2: econv_launch<2>(a, ctx->stream); break;
        case 3: econv_launch<3>(a, ctx->stream); break;
        case 4: econv_launch<4>(a, ctx->stream); break;
        case 5: econv_launch<5>(a, ctx->stream); break;
        case 6: econv_launch<6>(a, ctx->stream); break;
        case 7: econv_launch<7>(a, ctx->stream); break;
        case 8: econv_launch<8>(a, ctx->stream); break;
        case 9: econv_launch<9>(a, ctx->stream); break;
        case 10: econv_launch<10>(a, ctx->stream); break;
        default: econv_launch<11>(a, ctx->stream); break;
    }
    NEGF_LAUNCH_CHECK(ctx);
    return NEGF_OK;
}
