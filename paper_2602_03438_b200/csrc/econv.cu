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
// One CTA takes TE consecutive elements for ALL energies: rows of TE elements are read coalesced into
// shared memory as s[energy][element] (this IS the transposition: the FFT then runs along the energy axis
// with the element index across threads, conflict-free), zero-padded to L = 2^p >= 2 N_E - 1; radix-2
// decimation-in-frequency forward transforms of both operands (bit-reversed output), pointwise product,
// decimation-in-time inverse transform (natural output), scaled rows written back coalesced.  HBM-bound:
// 2 N_E + (2 N_E - 1) complex numbers per element, each touched once.
#include "common.cuh"

namespace {

constexpr int ECONV_NT = 256;
constexpr int ECONV_TILE = 2048;          // TE * L complex numbers per operand (32 KB): three CTAs per SM

struct EconvArgs {
    int ne, L, logL, te, lt; long long M;    // te = 2^lt elements per CTA
    int mode, conj2, bt;                   // bt = block size for transposing X2's blocks, 0 = none
    const cplx* X1; const cplx* X2; cplx* Y; cplx scale;
};

__global__ void __launch_bounds__(ECONV_NT) econv_kernel(EconvArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* sa = reinterpret_cast<cplx*>(smem_raw);          // [L][te]
    cplx* sb = sa + (size_t)a.L * a.te;                     // [L][te]
    cplx* tw = sb + (size_t)a.L * a.te;                     // [L/2]  exp(-2 pi i j / L)
    const int tid = threadIdx.x, te = a.te, lt = a.lt, tm = a.te - 1, L = a.L, ne = a.ne;
    const long long e0 = (long long)blockIdx.x * te;
    for (int j = tid; j < L / 2; j += ECONV_NT) {
        double sn, cs;
        sincospi(-2.0 * (double)j / (double)L, &sn, &cs);
        tw[j] = cmake(cs, sn);
    }
    // load, zero-padded; the second operand reversed in energy for a correlation
    for (int idx = tid; idx < L * te; idx += ECONV_NT) {
        const int k = idx >> lt, t = idx & tm;
        const long long el = e0 + t;
        cplx x = cmake(0.0, 0.0), y = x;
        if (k < ne && el < a.M) {
            x = a.X1[(size_t)k * a.M + el];
            long long el2 = el;
            if (a.bt) {                                     // (blk, i, j) -> (blk, j, i)
                if (a.M < 2147483647LL) {                   // 32-bit index arithmetic whenever it fits
                    const unsigned bt = (unsigned)a.bt, bb = bt * bt, eu = (unsigned)el, blk = eu / bb, r = eu % bb;
                    el2 = (long long)(blk * bb + (r % bt) * bt + r / bt);
                } else {
                    const long long bb = (long long)a.bt * a.bt, blk = el / bb, r = el % bb;
                    el2 = blk * bb + (r % a.bt) * a.bt + r / a.bt;
                }
            }
            const int k2 = a.mode ? ne - 1 - k : k;
            y = a.X2[(size_t)k2 * a.M + el2];
            if (a.conj2) y.y = -y.y;
        }
        sa[idx] = x; sb[idx] = y;
    }
    __syncthreads();
    // forward DIF, both operands: (p, p + h): x_p = a + b, x_{p+h} = (a - b) w^(j L / 2h), j = p mod h
    for (int lh = a.logL - 1, ls = 0; lh >= 0; lh--, ls++) {
        const int h = 1 << lh;
        for (int idx = tid; idx < (L >> 1) * te; idx += ECONV_NT) {
            const int bf = idx >> lt, t = idx & tm;
            const int j = bf & (h - 1), p = ((bf >> lh) << (lh + 1)) + j;
            const cplx w = tw[j << ls];
            cplx u = sa[p * te + t], v = sa[(p + h) * te + t];
            sa[p * te + t] = cadd(u, v); sa[(p + h) * te + t] = cmul(csub(u, v), w);
            u = sb[p * te + t]; v = sb[(p + h) * te + t];
            sb[p * te + t] = cadd(u, v); sb[(p + h) * te + t] = cmul(csub(u, v), w);
        }
        __syncthreads();
    }
    for (int idx = tid; idx < L * te; idx += ECONV_NT) sa[idx] = cmul(sa[idx], sb[idx]);
    __syncthreads();
    // inverse DIT on bit-reversed input: x_p = a + b conj(w)^(j L / 2h), x_{p+h} = a - (..)
    for (int lh = 0, ls = a.logL - 1; lh < a.logL; lh++, ls--) {
        const int h = 1 << lh;
        for (int idx = tid; idx < (L >> 1) * te; idx += ECONV_NT) {
            const int bf = idx >> lt, t = idx & tm;
            const int j = bf & (h - 1), p = ((bf >> lh) << (lh + 1)) + j;
            const cplx w = cconj(tw[j << ls]);
            const cplx u = sa[p * te + t], v = cmul(sa[(p + h) * te + t], w);
            sa[p * te + t] = cadd(u, v); sa[(p + h) * te + t] = csub(u, v);
        }
        __syncthreads();
    }
    const cplx sc = cmake(a.scale.x / L, a.scale.y / L);
    for (int idx = tid; idx < (2 * ne - 1) * te; idx += ECONV_NT) {
        const int m = idx >> lt, t = idx & tm;
        if (e0 + t < a.M) a.Y[(size_t)m * a.M + e0 + t] = cmul(sa[idx], sc);
    }
}

}  // namespace

extern "C" int negf_energy_convolve(negf_ctx* ctx, int n_energy, long long elems_per_energy, int transpose_block,
                                    const negf_c128* X1, const negf_c128* X2, int mode, int conj2, negf_c128 scale,
                                    negf_c128* Y) {
    if (!ctx || !X1 || !X2 || !Y || n_energy < 1 || elems_per_energy < 1 || (mode & ~1) || (conj2 & ~1)) return NEGF_EINVAL;
    if (transpose_block < 0 || (transpose_block > 0 && elems_per_energy % ((long long)transpose_block * transpose_block)))
        return NEGF_EINVAL;
    int L = 2, logL = 1;
    while (L < 2 * n_energy - 1) { L <<= 1; logL++; }
    if (L > ECONV_TILE) return NEGF_EUNSUPPORTED;          // N_E <= 1024
    EconvArgs a;
    a.ne = n_energy; a.L = L; a.logL = logL; a.te = ECONV_TILE / L; a.M = elems_per_energy;
    a.lt = 0; while ((1 << a.lt) < a.te) a.lt++;
    a.mode = mode; a.conj2 = conj2; a.bt = transpose_block;
    a.X1 = (const cplx*)X1; a.X2 = (const cplx*)X2; a.Y = (cplx*)Y; a.scale = cmake(scale.re, scale.im);
    const size_t smem = ((size_t)2 * ECONV_TILE + L / 2) * sizeof(cplx);
    static bool attr_done = false;
    if (!attr_done) {
        NEGF_CUDA_CHECK(ctx, cudaFuncSetAttribute(econv_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                  (int)(((size_t)2 * ECONV_TILE + ECONV_TILE / 2) * sizeof(cplx))));
        attr_done = true;
    }
    const long long ctas = (elems_per_energy + a.te - 1) / a.te;
    if (ctas > 2147483647LL) return NEGF_EUNSUPPORTED;
    ProfScope _ps(ctx, NEGF_PROF_ELEMENTWISE);
    econv_kernel<<<(unsigned)ctas, ECONV_NT, smem, ctx->stream>>>(a);
    NEGF_LAUNCH_CHECK(ctx);
    return NEGF_OK;
}
