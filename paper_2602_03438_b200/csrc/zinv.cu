// K1: batched in-place complex inverse with partial pivoting.
//
// Every g_i = (A_ii - A_{i,i-1} g_{i-1} A_{i-1,i})^-1 of the RGF forward sweep (
// SURVEY.md 8(a) S3) and every g = a_b^-1 of the Sancho-Rubio doubling is one
// call of this file.
//
//  * b <= SMALL_MAX: one CTA per matrix, whole matrix in shared memory, in-place Gauss-Jordan
//    with row pivoting on |re|+|im| (izamax convention), column permutation undone at the end.
//  * larger b: BLOCKED in-place Gauss-Jordan, panel width w <= 32:
//      1. the panel (rows >= k0) is LU-factorised with partial pivoting by a thread-block
//         CLUSTER that holds the tall panel in distributed shared memory (up to 8 CTAs x 200 KB);
//         every column costs ONE cluster barrier: before it each CTA pushes its best pivot
//         candidate (value, row index, row content) and CTA 0 the current diagonal row into all
//         CTAs' buffers through DSMEM, after it everybody knows the pivot and already owns the
//         two rows to exchange;
//      2. row swaps are applied to the rest of the matrix, the pivot rows R are moved to scratch
//         and zeroed;
//      3. the panel is finalised to P' = [-T Dinv ; Dinv ; -L21 L11^-1] with two small GEMMs;
//      4. ONE rank-w GEMM per side updates all other columns: M += P' R  (K2 kernel, DMMA).
//    Cost b^3 complex multiply-adds = 8 b^3 flops = 1 U, same as getrf + getri, but every
//    trailing update is a full-height uniform GEMM.  Pivoting is partial pivoting among the
//    not-yet-eliminated rows, exactly as in LU.
#include <cooperative_groups.h>

#include "common.cuh"

namespace cg = cooperative_groups;

namespace {

constexpr int SMALL_MAX = 96;      // b*b*16 B <= 147 KB
constexpr int PW = 32;             // max panel width (one lane per panel column)
constexpr int CMAX = 8;            // portable cluster size
constexpr int PANEL_SMEM_ROWS_BYTES = 176 * 1024;   // + 9 KB exchange buffers + 33 KB static < 227 KB

// ------------------------------------------------------------------------------------------------
// small path: REGISTER-resident Gauss-Jordan, one CTA of 8 warps per matrix (b <= 96).
//   * warp w owns the columns j = w + 8 c (c < CB), lane l the rows i = l + 32 r (r < RB): the
//     whole matrix lives in registers (RB x CB elements per thread);
//   * the pivot search of column k is done by its owner warp alone with three redux.sync on the
//     bit pattern of |re|+|im| (monotone for non-negative doubles), which then publishes the
//     multiplier column, the pivot index and 1/pivot to shared memory;
//   * ONE block barrier per column; the two rows that trade places travel inside each warp
//     through a per-warp shared-memory line (no block-level traffic);
//   * look-ahead: the owner of column k+1 updates that column first, searches its pivot and
//     publishes it BEFORE finishing its update for column k, so the barrier of column k+1 never
//     waits for a pivot search;
//   * the rank-1 update runs out of registers at the DFMA rate (= the DMMA rate on sm_100).
// Rows/columns >= b are padded with the identity and never reached.
// ------------------------------------------------------------------------------------------------
constexpr int GJ_NW = 8;


__device__ __forceinline__ cplx crecip_fast(cplx a) {      // pivots are O(1): no overflow guard needed
    const double inv = 1.0 / fma(a.x, a.x, a.y * a.y);
    return cmake(a.x * inv, -a.y * inv);
}

struct GjShared {            // pointers into the kernel's shared memory
    cplx* colbuf;            // [2][NR]
    cplx* wrow;              // this warp's [2][2][CB]
    cplx* s_d; int* s_p; int* piv; int* s_sing;
};

// pivot search + publication of column kn, held in slot C of the calling (owner) warp
template <int RB, int CB, int C>
__device__ __forceinline__ void gj_owner(const cplx (&m)[RB][CB], const GjShared& sh, int kn, int b, int lane) {
    constexpr int NR = RB * 32;
    const int parn = kn & 1;
    unsigned long long key = 0ull;
    int bi = 0x7fffffff;
#pragma unroll
    for (int r = 0; r < RB; r++) {
        const int i = lane + 32 * r;
        sh.colbuf[parn * NR + i] = m[r][C];
        if (i >= kn && i < b) {
            const unsigned long long kq = (unsigned long long)__double_as_longlong(cabs1(m[r][C]));
            if (bi == 0x7fffffff || kq > key) { key = kq; bi = i; }
        }
    }
    const bool has = bi != 0x7fffffff;
    const unsigned hi = __reduce_max_sync(0xffffffffu, has ? (unsigned)(key >> 32) : 0u);
    const bool mh = has && (unsigned)(key >> 32) == hi;
    const unsigned lo = __reduce_max_sync(0xffffffffu, mh ? (unsigned)key : 0u);
    const bool ml = mh && (unsigned)key == lo;
    const unsigned p = __reduce_min_sync(0xffffffffu, ml ? (unsigned)bi : 0x7fffffffu);
    cplx pv = cmake(0.0, 0.0);
#pragma unroll
    for (int r = 0; r < RB; r++) if (lane + 32 * r == (int)p) pv = m[r][C];
    pv.x = __shfl_sync(0xffffffffu, pv.x, p & 31);
    pv.y = __shfl_sync(0xffffffffu, pv.y, p & 31);
    const bool sing = (hi == 0u && lo == 0u);
    if (lane == 0) {
        sh.s_p[parn] = (int)p; sh.piv[kn] = (int)p;
        sh.s_d[parn] = sing ? cmake(1.0, 0.0) : crecip_fast(pv);
        if (sing && *sh.s_sing == 0) *sh.s_sing = kn + 1;
    }
}

// Rank-1 update of column slot C: m[:, C] -= mult * sr.  The special rows/columns were prepared by
// the caller so that this one formula is right everywhere (pivot row: m = 0, mult = -1 -> sr;
// pivot column: m = 0, sr = 1/pivot -> -mult/pivot).
template <int RB, int CB, int C>
__device__ __forceinline__ void gj_update(cplx (&m)[RB][CB], const cplx (&mult)[RB], const cplx (&sr)[CB]) {
#pragma unroll
    for (int r = 0; r < RB; r++) cfms(m[r][C], mult[r], sr[C]);
}

template <int RB, int CB, int C>
__device__ __forceinline__ void gj_update_rest(cplx (&m)[RB][CB], const cplx (&mult)[RB], const cplx (&sr)[CB], int done) {
    if constexpr (C < CB) {
        if (C != done) gj_update<RB, CB, C>(m, mult, sr);
        gj_update_rest<RB, CB, C + 1>(m, mult, sr, done);
    }
}

// all columns k = CK*8 + wk, wk < 8, then recurse to CK + 1
template <int RB, int CB, int CK>
__device__ __forceinline__ void gj_columns(cplx (&m)[RB][CB], const GjShared& sh, int b, int warp, int lane) {
    if constexpr (CK < CB) {
        constexpr int NR = RB * 32;
        constexpr int CN = (CK + 1 < CB) ? CK + 1 : CK;
#pragma unroll 1
        for (int wk = 0; wk < GJ_NW; wk++) {
            const int k = CK * GJ_NW + wk;
            if (k >= b) break;
            const int par = k & 1;
            __syncthreads();
            const int p = sh.s_p[par];
            const cplx d = sh.s_d[par];
            cplx* wr = sh.wrow + par * 2 * CB;
            // the two rows that trade places, through this warp's shared-memory line
#pragma unroll
            for (int r = 0; r < RB; r++) {
                const int i = lane + 32 * r;
                if (i == p) {
#pragma unroll
                    for (int c = 0; c < CB; c++) wr[c] = m[r][c];
                }
                if (i == k && p != k) {
#pragma unroll
                    for (int c = 0; c < CB; c++) wr[CB + c] = m[r][c];
                }
            }
            __syncwarp();
            cplx mult[RB];
#pragma unroll
            for (int r = 0; r < RB; r++) {
                const int i = lane + 32 * r;
                mult[r] = sh.colbuf[par * NR + ((i == p) ? k : i)];   // row p inherits old row k's multiplier
                if (i == p && p != k) {
#pragma unroll
                    for (int c = 0; c < CB; c++) m[r][c] = wr[CB + c];
                }
                if (i == k) {
                    mult[r] = cmake(-1.0, 0.0);
#pragma unroll
                    for (int c = 0; c < CB; c++) m[r][c] = cmake(0.0, 0.0);
                }
            }
            cplx sr[CB];
#pragma unroll
            for (int c = 0; c < CB; c++) sr[c] = cmul(wr[c], d);
            if (warp == wk) {            // this warp's slot CK IS column k
                sr[CK] = d;
#pragma unroll
                for (int r = 0; r < RB; r++) m[r][CK] = cmake(0.0, 0.0);
            }
            // look-ahead: the owner of column k+1 brings that column up to date and publishes it first
            int done = -1;
            if (k + 1 < b && warp == ((wk + 1) & (GJ_NW - 1))) {
                if (wk < GJ_NW - 1) {
                    gj_update<RB, CB, CK>(m, mult, sr);
                    gj_owner<RB, CB, CK>(m, sh, k + 1, b, lane);
                    done = CK;
                } else if (CK + 1 < CB) {
                    gj_update<RB, CB, CN>(m, mult, sr);
                    gj_owner<RB, CB, CN>(m, sh, k + 1, b, lane);
                    done = CN;
                }
            }
            gj_update_rest<RB, CB, 0>(m, mult, sr, done);
        }
        gj_columns<RB, CB, CK + 1>(m, sh, b, warp, lane);
    }
}

template <int RB, int CB>
__global__ void __launch_bounds__(GJ_NW * 32) gj_reg_kernel(cplx* A, long long sA, int b, int* info, int code,
                                                            const int* skip) {
    constexpr int NR = RB * 32, NC = CB * GJ_NW;
    const int e = blockIdx.x;
    if (skip && skip[e]) return;
    __shared__ cplx colbuf[2 * NR];
    __shared__ cplx wrow[GJ_NW][2 * 2 * CB];     // [warp][parity][pivot row | row k][slot]
    __shared__ cplx s_d[2];
    __shared__ int s_p[2];
    __shared__ int piv[NC];
    __shared__ int dest[NC];
    __shared__ int s_sing;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    cplx* g = A + (size_t)e * sA;
    cplx m[RB][CB];
#pragma unroll
    for (int r = 0; r < RB; r++)
#pragma unroll
        for (int c = 0; c < CB; c++) {
            const int i = lane + 32 * r, j = warp + GJ_NW * c;
            m[r][c] = (i < b && j < b) ? g[(size_t)i * b + j] : cmake(i == j ? 1.0 : 0.0, 0.0);
        }
    if (tid == 0) s_sing = 0;
    __syncthreads();
    GjShared sh{colbuf, wrow[warp], s_d, s_p, piv, &s_sing};
    if (warp == 0) gj_owner<RB, CB, 0>(m, sh, 0, b, lane);
    gj_columns<RB, CB, 0>(m, sh, b, warp, lane);
    __syncthreads();
    // A^-1 = (P A)^-1 P: column j of the result is column src[j] of M, src = the recorded swaps
    // applied in reverse order to the identity; every thread scatters its columns to src^-1.
    if (tid == 0) {
        for (int c = 0; c < b; c++) dest[c] = c;
        for (int k = b - 1; k >= 0; k--) {
            const int p = piv[k];
            if (p != k) { int t = dest[k]; dest[k] = dest[p]; dest[p] = t; }
        }
        for (int c = 0; c < b; c++) piv[dest[c]] = c;     // piv now holds src^-1
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < RB; r++)
#pragma unroll
        for (int c = 0; c < CB; c++) {
            const int i = lane + 32 * r, j = warp + GJ_NW * c;
            if (i < b && j < b) g[(size_t)i * b + piv[j]] = m[r][c];
        }
    if (tid == 0 && s_sing && info) info[e] = code > 0 ? code : s_sing;
}

// ------------------------------------------------------------------------------------------------
// blocked path, step 1: cluster panel LU with partial pivoting
// ------------------------------------------------------------------------------------------------
struct Cand { double val; int row; int pad; };

struct PanelArgs {
    cplx* A; long long sA; int b, k0, w, slab;
    int* ipiv;            // [batch][b] global row index chosen for column k
    cplx* Dinv;           // [batch][PW*PW] (ld = w)  (L11 U11)^-1
    cplx* Linv;           // [batch][PW*PW] (ld = w)  L11^-1
    int* info; int code; const int* skip;
};

constexpr int PANEL_NT = 512;

__global__ void __launch_bounds__(PANEL_NT, 1) gj_panel_cluster_kernel(PanelArgs a) {
    cg::cluster_group cluster = cg::this_cluster();
    const int rank = (int)cluster.block_rank();
    const int C = (int)cluster.num_blocks();
    const int e = blockIdx.y;
    if (a.skip && a.skip[e]) return;              // uniform over the cluster
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int w = a.w, b = a.b, k0 = a.k0, slab = a.slab;
    cplx* P = reinterpret_cast<cplx*>(smem_raw);                    // [slab][w]
    cplx* candrow = P + (size_t)slab * w;                           // [2][CMAX][PW]
    cplx* diagrow = candrow + 2 * CMAX * PW;                        // [2][PW]
    Cand* cand = reinterpret_cast<Cand*>(diagrow + 2 * PW);         // [2][CMAX]
    __shared__ double red_val[PANEL_NT / 32];
    __shared__ int red_idx[PANEL_NT / 32];
    __shared__ int s_best;

    const int rows_total = b - k0;
    const int r_lo = rank * slab;
    const int nloc = max(0, min(rows_total, r_lo + slab) - r_lo);
    cplx* g = a.A + (size_t)e * a.sA + (size_t)k0 * b + k0;       // panel origin
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int NW = PANEL_NT / 32;

    for (int idx = tid; idx < nloc * w; idx += PANEL_NT) {
        int r = idx / w, j = idx % w;
        P[r * w + j] = g[(size_t)(r_lo + r) * b + j];
    }
    __syncthreads();

    for (int j = 0; j < w; j++) {
        const int par = j & 1;
        // local pivot candidate among my rows with global candidate index >= j
        double best = -1.0; int bi = -1;
        for (int r = tid; r < nloc; r += PANEL_NT) {
            if (r_lo + r >= j) {
                double v = cabs1(P[r * w + j]);
                if (v > best) { best = v; bi = r; }
            }
        }
        for (int o = 16; o > 0; o >>= 1) {
            double ov = __shfl_down_sync(0xffffffffu, best, o);
            int oi = __shfl_down_sync(0xffffffffu, bi, o);
            if (ov > best || (ov == best && oi >= 0 && (bi < 0 || oi < bi))) { best = ov; bi = oi; }
        }
        if (lane == 0) { red_val[warp] = best; red_idx[warp] = bi; }
        __syncthreads();
        if (warp == 0) {
            best = lane < NW ? red_val[lane] : -1.0;
            bi = lane < NW ? red_idx[lane] : -1;
            for (int o = 16; o > 0; o >>= 1) {
                double ov = __shfl_down_sync(0xffffffffu, best, o);
                int oi = __shfl_down_sync(0xffffffffu, bi, o);
                if (ov > best || (ov == best && oi >= 0 && (bi < 0 || oi < bi))) { best = ov; bi = oi; }
            }
            best = __shfl_sync(0xffffffffu, best, 0);
            bi = __shfl_sync(0xffffffffu, bi, 0);
            // push (value, row, row content) to every CTA of the cluster; CTA 0 also the diagonal row
            cplx myrow = (bi >= 0 && lane < w) ? P[bi * w + lane] : cmake(0.0, 0.0);
            cplx drow = (rank == 0 && lane < w) ? P[j * w + lane] : cmake(0.0, 0.0);
            for (int q = 0; q < C; q++) {
                cplx* rc = cluster.map_shared_rank(candrow, q);
                if (lane < w) rc[(par * CMAX + rank) * PW + lane] = myrow;
                if (rank == 0 && lane < w) cluster.map_shared_rank(diagrow, q)[par * PW + lane] = drow;
                if (lane == 0) {
                    Cand c; c.val = best; c.row = bi >= 0 ? r_lo + bi : -1; c.pad = 0;
                    cluster.map_shared_rank(cand, q)[par * CMAX + rank] = c;
                }
            }
        }
        cluster.sync();
        // everybody picks the same winner
        if (tid == 0) {
            int wq = -1; double wv = -1.0; int wr = 0x7fffffff;
            for (int q = 0; q < C; q++) {
                Cand c = cand[par * CMAX + q];
                if (c.row >= 0 && (c.val > wv || (c.val == wv && c.row < wr))) { wv = c.val; wq = q; wr = c.row; }
            }
            s_best = wq;
            if (rank == 0) {
                a.ipiv[(size_t)e * b + k0 + j] = k0 + wr;
                if (!(wv > 0.0) && a.info && a.info[e] == 0) a.info[e] = a.code > 0 ? a.code : (k0 + j + 1);
            }
        }
        __syncthreads();
        const int wq = s_best;
        const int prow = cand[par * CMAX + wq].row;                 // global candidate index of the pivot row
        const double pval = cand[par * CMAX + wq].val;
        const cplx* pr = candrow + (par * CMAX + wq) * PW;          // pivot row content
        // exchange rows j <-> prow
        if (prow != j && warp == 0 && lane < w) {
            if (prow >= r_lo && prow < r_lo + nloc) P[(prow - r_lo) * w + lane] = diagrow[par * PW + lane];
        }
        if (rank == 0 && warp == 1 && lane < w) P[j * w + lane] = pr[lane];
        __syncthreads();
        // eliminate below: rows with candidate index > j
        cplx pv = pr[j];
        cplx rinv = (pval > 0.0) ? crecip(pv) : cmake(0.0, 0.0);
        cplx pvl = lane < w ? pr[lane] : cmake(0.0, 0.0);
        for (int r = warp; r < nloc; r += NW) {
            if (r_lo + r > j) {
                cplx l = cmul(P[r * w + j], rinv);
                __syncwarp();
                if (lane == j) P[r * w + j] = l;
                else if (lane > j && lane < w) { cplx v = P[r * w + lane]; cfms(v, l, pvl); P[r * w + lane] = v; }
            }
        }
        __syncthreads();
    }

    // CTA 0: L11^-1 and (L11 U11)^-1 from the w x w diagonal block, one thread per column
    if (rank == 0) {
        __shared__ cplx Li[PW * PW];
        __shared__ cplx sUi[PW * PW];
        // Linv (unit lower): solve L X = I column by column
        if (tid < w) {
            int c = tid;
            for (int r = 0; r < w; r++) {
                cplx s = (r == c) ? cmake(1.0, 0.0) : cmake(0.0, 0.0);
                for (int k = c; k < r; k++) cfms(s, P[r * w + k], Li[k * PW + c]);
                Li[r * PW + c] = (r < c) ? cmake(0.0, 0.0) : s;
            }
        } else if (tid >= 32 && tid < 32 + w) {
            // Uinv: solve U X = I column by column (back substitution)
            int c = tid - 32;
            for (int r = w - 1; r >= 0; r--) {
                cplx s = (r == c) ? cmake(1.0, 0.0) : cmake(0.0, 0.0);
                for (int k = r + 1; k <= c; k++) cfms(s, P[r * w + k], sUi[k * PW + c]);
                cplx ur = P[r * w + r];
                cplx inv = (ur.x == 0.0 && ur.y == 0.0) ? cmake(0.0, 0.0) : crecip(ur);
                sUi[r * PW + c] = (r > c) ? cmake(0.0, 0.0) : cmul(s, inv);
            }
        }
        __syncthreads();
        cplx* gD = a.Dinv + (size_t)e * PW * PW;
        cplx* gL = a.Linv + (size_t)e * PW * PW;
        for (int idx = tid; idx < w * w; idx += PANEL_NT) {
            int r = idx / w, c = idx % w;
            cplx s = cmake(0.0, 0.0);
            for (int k = max(r, c); k < w; k++) cfma(s, sUi[r * PW + k], Li[k * PW + c]);
            gD[r * w + c] = s;
            gL[r * w + c] = Li[r * PW + c];
        }
    }
    // write the factored panel back (L21 below, L11\U11 in the diagonal block)
    for (int idx = tid; idx < nloc * w; idx += PANEL_NT) {
        int r = idx / w, j = idx % w;
        g[(size_t)(r_lo + r) * b + j] = P[r * w + j];
    }
    cluster.sync();   // nobody exits while remote shared memory may still be targeted
}

// ------------------------------------------------------------------------------------------------
// step 1, register-resident variant (tall panels up to 8 x 256 rows): every thread owns ONE row of
// the width-32 panel in registers, a cluster of C CTAs covers the rows >= k0.  Per column: one
// redux-based candidate per CTA, one DSMEM exchange (candidate value, row index, row content and
// the current diagonal row) and one cluster barrier; the elimination runs out of registers.  The
// kernel also finishes the panel in place: rows below the diagonal block leave as -L21 L11^-1,
// the diagonal block as (L11 U11)^-1, so the trailing GEMM reads P' straight from A's columns.
// ------------------------------------------------------------------------------------------------
struct RegPanelSmem {
    cplx candrow[2][CMAX][PW];
    cplx diagrow[2][PW];
    cplx rowstage[PW];
    cplx drowstage[PW];
    cplx Dm[PW * PW];      // factored diagonal block L11 \ U11
    cplx Li[PW * PW];      // L11^-1 (every CTA gets a copy)
    cplx Ui[PW * PW];      // U11^-1 (CTA 0)
    unsigned long long red_key[8];
    int red_row[8];
    unsigned long long cand_key[2][CMAX];
    int cand_row[2][CMAX];
};

template <int NT>
__global__ void __launch_bounds__(NT) gj_panel_reg_kernel(PanelArgs a) {
    cg::cluster_group cluster = cg::this_cluster();
    const int rank = (int)cluster.block_rank();
    const int C = (int)cluster.num_blocks();
    const int e = blockIdx.y;
    if (a.skip && a.skip[e]) return;              // uniform over the cluster
    extern __shared__ __align__(16) unsigned char smem_raw[];
    RegPanelSmem& S = *reinterpret_cast<RegPanelSmem*>(smem_raw);
    const int w = a.w, b = a.b, k0 = a.k0;
    const int rows_total = b - k0;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int gr = rank * NT + tid;               // candidate row index (global row k0 + gr)
    const bool valid = gr < rows_total;
    cplx* g = a.A + (size_t)e * a.sA + (size_t)k0 * b + k0;       // panel origin
    cplx P[PW];
#pragma unroll
    for (int c = 0; c < PW; c++) P[c] = (valid && c < w) ? g[(size_t)gr * b + c] : cmake(0.0, 0.0);
    constexpr int NONE = 0x7fffffff;

    // The column loop is deliberately NOT unrolled (a fully unrolled body is ~13k instructions that
    // each run once: ncu showed 47 % of the stall cycles in instruction fetch); the register row
    // is addressed with compile-time indices and the current column is picked by predication.
#pragma unroll 1
    for (int j = 0; j < w; j++) {
        const int par = j & 1;
        cplx pj = cmake(0.0, 0.0);
#pragma unroll
        for (int c = 0; c < PW; c++) if (c == j) pj = P[c];
        // CTA candidate: largest |re|+|im| among my rows with index >= j (smallest row on ties)
        const bool has = valid && gr >= j;
        const unsigned long long key = has ? (unsigned long long)__double_as_longlong(cabs1(pj)) : 0ull;
        const unsigned hi = __reduce_max_sync(0xffffffffu, has ? (unsigned)(key >> 32) : 0u);
        const bool mh = has && (unsigned)(key >> 32) == hi;
        const unsigned lo = __reduce_max_sync(0xffffffffu, mh ? (unsigned)key : 0u);
        const bool ml = mh && (unsigned)key == lo;
        const unsigned wrow = __reduce_min_sync(0xffffffffu, ml ? (unsigned)gr : (unsigned)NONE);
        if (lane == 0) { S.red_key[warp] = ((unsigned long long)hi << 32) | lo; S.red_row[warp] = (int)wrow; }
        __syncthreads();
        unsigned long long bk = 0ull; int br = NONE;
#pragma unroll
        for (int q = 0; q < NT / 32; q++) {
            const unsigned long long k2 = S.red_key[q]; const int r2 = S.red_row[q];
            if (r2 != NONE && (br == NONE || k2 > bk || (k2 == bk && r2 < br))) { bk = k2; br = r2; }
        }
        if (gr == br) {
#pragma unroll
            for (int c = 0; c < PW; c++) S.rowstage[c] = P[c];
        }
        if (rank == 0 && tid == j) {
#pragma unroll
            for (int c = 0; c < PW; c++) S.drowstage[c] = P[c];
        }
        __syncthreads();
        if (warp == 0) {       // push (value, row, row content) to every CTA; CTA 0 also the diagonal row
            const cplx myrow = S.rowstage[lane];
            const cplx drow = S.drowstage[lane];
            for (int q = 0; q < C; q++) {
                RegPanelSmem* R = cluster.map_shared_rank(&S, q);
                R->candrow[par][rank][lane] = myrow;
                if (rank == 0) R->diagrow[par][lane] = drow;
                if (lane == 0) { R->cand_key[par][rank] = bk; R->cand_row[par][rank] = br; }
            }
        }
        cluster.sync();
        // everybody picks the same winner
        int wq = 0, prow = NONE; unsigned long long wk = 0ull;
        for (int q = 0; q < C; q++) {
            const unsigned long long k2 = S.cand_key[par][q]; const int r2 = S.cand_row[par][q];
            if (r2 != NONE && (prow == NONE || k2 > wk || (k2 == wk && r2 < prow))) { wk = k2; prow = r2; wq = q; }
        }
        const bool sing = (prow == NONE) || wk == 0ull;
        if (prow == NONE) prow = j;
        if (rank == 0 && tid == 0) {
            a.ipiv[(size_t)e * b + k0 + j] = k0 + prow;
            if (sing && a.info && a.info[e] == 0) a.info[e] = a.code > 0 ? a.code : (k0 + j + 1);
        }
        const cplx* pr = S.candrow[par][wq];
        // exchange rows j <-> prow
        if (valid && gr == prow && prow != j) {
#pragma unroll
            for (int c = 0; c < PW; c++) P[c] = S.diagrow[par][c];
        }
        if (rank == 0 && tid == j && prow != j) {
#pragma unroll
            for (int c = 0; c < PW; c++) P[c] = pr[c];
        }
        // eliminate below
        if (valid && gr > j) {
            cplx mine = cmake(0.0, 0.0);
#pragma unroll
            for (int c = 0; c < PW; c++) if (c == j) mine = P[c];
            const cplx rinv = sing ? cmake(0.0, 0.0) : crecip(pr[j]);
            const cplx l = cmul(mine, rinv);
#pragma unroll
            for (int c = 0; c < PW; c++) {
                if (c == j) P[c] = l;
                else if (c > j) cfms(P[c], l, pr[c]);
            }
        }
    }

    // CTA 0: L11^-1 and U11^-1 from the w x w diagonal block, one thread per column; then
    // (L11 U11)^-1 = U11^-1 L11^-1; L11^-1 goes to every CTA of the cluster.
    if (rank == 0) {
        for (int idx = tid; idx < PW * PW; idx += NT) { S.Li[idx] = cmake(0.0, 0.0); S.Ui[idx] = cmake(0.0, 0.0); }
        if (tid < w) {
#pragma unroll
            for (int c = 0; c < PW; c++) S.Dm[tid * PW + c] = P[c];
        }
        __syncthreads();
        if (tid < w) {
            const int c = tid;
            for (int r = 0; r < w; r++) {
                cplx s = (r == c) ? cmake(1.0, 0.0) : cmake(0.0, 0.0);
                for (int k = c; k < r; k++) cfms(s, S.Dm[r * PW + k], S.Li[k * PW + c]);
                S.Li[r * PW + c] = (r < c) ? cmake(0.0, 0.0) : s;
            }
        } else if (tid >= 32 && tid < 32 + w) {
            const int c = tid - 32;
            for (int r = w - 1; r >= 0; r--) {
                cplx s = (r == c) ? cmake(1.0, 0.0) : cmake(0.0, 0.0);
                for (int k = r + 1; k <= c; k++) cfms(s, S.Dm[r * PW + k], S.Ui[k * PW + c]);
                const cplx ur = S.Dm[r * PW + r];
                const cplx inv = (ur.x == 0.0 && ur.y == 0.0) ? cmake(0.0, 0.0) : crecip(ur);
                S.Ui[r * PW + c] = (r > c) ? cmake(0.0, 0.0) : cmul(s, inv);
            }
        }
        __syncthreads();
        cplx* gD = a.Dinv + (size_t)e * PW * PW;
        for (int idx = tid; idx < w * w; idx += NT) {
            const int r = idx / w, c = idx % w;
            cplx s = cmake(0.0, 0.0);
            for (int k = max(r, c); k < w; k++) cfma(s, S.Ui[r * PW + k], S.Li[k * PW + c]);
            gD[r * w + c] = s;
            g[(size_t)r * b + c] = s;                       // diagonal block of P' in place
        }
        for (int idx = tid; idx < PW * PW; idx += NT) {
            const cplx v = S.Li[idx];
            for (int q = 1; q < C; q++) cluster.map_shared_rank(&S, q)->Li[idx] = v;
        }
    }
    cluster.sync();
    // rows below the diagonal block: P' = -L21 L11^-1, written in place
    if (valid && gr >= w) {
        cplx* out = g + (size_t)gr * b;
#pragma unroll 1
        for (int c = 0; c < w; c++) {
            cplx acc = cmake(0.0, 0.0);
#pragma unroll
            for (int k = 0; k < PW; k++) cfms(acc, P[k], S.Li[k * PW + c]);    // Li[k][c] = 0 for k < c and k >= w
            out[c] = acc;
        }
    }
    cluster.sync();   // nobody exits while remote shared memory may still be targeted
}

// ------------------------------------------------------------------------------------------------
// step 2: apply the panel's row swaps to all other columns; move pivot rows to R and zero them
// ------------------------------------------------------------------------------------------------
// pivots p0 .. p0+np-1; columns [clo, chi) except [xlo, xhi)
__global__ void gj_swap_extract_kernel(cplx* A, long long sA, int b, int p0, int np, int clo, int chi, int xlo,
                                       int xhi, const int* ipiv, cplx* R /*[batch][np][b]*/, const int* skip) {
    const int e = blockIdx.y;
    if (skip && skip[e]) return;
    int c = clo + blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= chi || (c >= xlo && c < xhi)) return;
    cplx* g = A + (size_t)e * sA;
    const int* pv = ipiv + (size_t)e * b + p0;
    for (int j = 0; j < np; j++) {
        int p = pv[j];
        if (p != p0 + j) {
            cplx t = g[(size_t)(p0 + j) * b + c];
            g[(size_t)(p0 + j) * b + c] = g[(size_t)p * b + c];
            g[(size_t)p * b + c] = t;
        }
    }
    cplx* r = R + (size_t)e * np * b;
    for (int j = 0; j < np; j++) {
        r[(size_t)j * b + c] = g[(size_t)(p0 + j) * b + c];
        g[(size_t)(p0 + j) * b + c] = cmake(0.0, 0.0);
    }
}

// copy the finalised panel Pbuf [b][w] into columns [k0, k0+w) of A
__global__ void gj_panel_store_kernel(cplx* A, long long sA, int b, int k0, int w, const cplx* Pbuf,
                                      const cplx* Dinv, const int* skip) {
    const int e = blockIdx.y;
    if (skip && skip[e]) return;
    int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= b * w) return;
    int r = idx / w, j = idx % w;
    cplx v = (r >= k0 && r < k0 + w) ? Dinv[(size_t)e * PW * PW + (r - k0) * w + j]
                                     : Pbuf[(size_t)e * b * w + idx];
    A[(size_t)e * sA + (size_t)r * b + k0 + j] = v;
}
// copy Dinv into rows [k0,k0+w) of Pbuf so the big GEMM sees the complete P'
__global__ void gj_pbuf_diag_kernel(cplx* Pbuf, int b, int k0, int w, const cplx* Dinv, const int* skip) {
    const int e = blockIdx.y;
    if (skip && skip[e]) return;
    int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= w * w) return;
    Pbuf[(size_t)e * b * w + (size_t)k0 * w + idx] = Dinv[(size_t)e * PW * PW + idx];
}

// final column permutation: idx[] from the recorded swaps, then a row-wise gather through smem
__global__ void gj_colperm_kernel(cplx* A, long long sA, int b, const int* ipiv, int* idxbuf, const int* skip) {
    const int e = blockIdx.y;
    if (skip && skip[e]) return;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* row = reinterpret_cast<cplx*>(smem_raw);
    int* idx = idxbuf + (size_t)e * b;
    // idx was computed by gj_permidx_kernel
    cplx* g = A + (size_t)e * sA;
    for (int r = blockIdx.x; r < b; r += gridDim.x) {
        for (int c = threadIdx.x; c < b; c += blockDim.x) row[c] = g[(size_t)r * b + c];
        __syncthreads();
        for (int c = threadIdx.x; c < b; c += blockDim.x) g[(size_t)r * b + c] = row[idx[c]];
        __syncthreads();
    }
}
__global__ void gj_permidx_kernel(int b, const int* ipiv, int* idxbuf, const int* skip) {
    const int e = blockIdx.x;
    if (skip && skip[e]) return;
    extern __shared__ int sidx[];
    for (int c = threadIdx.x; c < b; c += blockDim.x) sidx[c] = c;
    __syncthreads();
    if (threadIdx.x == 0) {
        const int* pv = ipiv + (size_t)e * b;
        for (int k = b - 1; k >= 0; k--) {
            int p = pv[k];
            if (p != k) { int t = sidx[k]; sidx[k] = sidx[p]; sidx[p] = t; }
        }
    }
    __syncthreads();
    for (int c = threadIdx.x; c < b; c += blockDim.x) idxbuf[(size_t)e * b + c] = sidx[c];
}

constexpr int OUTER_NB = 128;      // outer block of the two-level blocked Gauss-Jordan

struct InvWs {
    cplx* Rout;   // [batch][OUTER_NB][b]  pivot rows of an outer block
    cplx* R;      // [batch][PW][b]
    cplx* Pbuf;   // [batch][b][PW]
    cplx* Dinv;   // [batch][PW*PW]
    cplx* Linv;   // [batch][PW*PW]
    int* ipiv;    // [batch][b]
    int* idx;     // [batch][b]
};
InvWs carve(void* ws, int b, int batch) {
    InvWs o;
    unsigned char* p = (unsigned char*)ws;
    o.Rout = (cplx*)p; p += align_up((size_t)batch * OUTER_NB * b * sizeof(cplx), 256);
    o.R = (cplx*)p;    p += align_up((size_t)batch * PW * b * sizeof(cplx), 256);
    o.Pbuf = (cplx*)p; p += align_up((size_t)batch * PW * b * sizeof(cplx), 256);
    o.Dinv = (cplx*)p; p += align_up((size_t)batch * PW * PW * sizeof(cplx), 256);
    o.Linv = (cplx*)p; p += align_up((size_t)batch * PW * PW * sizeof(cplx), 256);
    o.ipiv = (int*)p;  p += align_up((size_t)batch * b * sizeof(int), 256);
    o.idx = (int*)p;
    return o;
}

}  // namespace

size_t zinv_workspace_bytes(int b, int batch) {
    if (b <= SMALL_MAX) return 256;
    return align_up((size_t)batch * OUTER_NB * b * sizeof(cplx), 256) +
           2 * align_up((size_t)batch * PW * b * sizeof(cplx), 256) +
           2 * align_up((size_t)batch * PW * PW * sizeof(cplx), 256) +
           2 * align_up((size_t)batch * b * sizeof(int), 256);
}

int zinv_launch(negf_ctx* ctx, int b, cplx* A, long long sA, int batch, void* ws, int* info,
                int info_code, const int* skip) {
    ProfScope _ps(ctx, NEGF_PROF_INVERSE);
    if (b <= 0 || batch <= 0) return NEGF_OK;
    if (b <= SMALL_MAX) {
        if (b <= 16)      gj_reg_kernel<1, 2><<<batch, GJ_NW * 32, 0, ctx->stream>>>(A, sA, b, info, info_code, skip);
        else if (b <= 32) gj_reg_kernel<1, 4><<<batch, GJ_NW * 32, 0, ctx->stream>>>(A, sA, b, info, info_code, skip);
        else if (b <= 48) gj_reg_kernel<2, 6><<<batch, GJ_NW * 32, 0, ctx->stream>>>(A, sA, b, info, info_code, skip);
        else if (b <= 64) gj_reg_kernel<2, 8><<<batch, GJ_NW * 32, 0, ctx->stream>>>(A, sA, b, info, info_code, skip);
        else if (b <= 80) gj_reg_kernel<3, 10><<<batch, GJ_NW * 32, 0, ctx->stream>>>(A, sA, b, info, info_code, skip);
        else              gj_reg_kernel<3, 12><<<batch, GJ_NW * 32, 0, ctx->stream>>>(A, sA, b, info, info_code, skip);
        NEGF_LAUNCH_CHECK(ctx);
        return NEGF_OK;
    }
    if (batch > 65535) return NEGF_EUNSUPPORTED;
    if (!ws) return NEGF_ENOWORKSPACE;
    InvWs W = carve(ws, b, batch);
    // panel width: the widest of 32/16/8 whose tall panel fits 8 CTAs of shared memory
    int w = PW;
    while (w > 8 && (size_t)((b + CMAX - 1) / CMAX) * w * sizeof(cplx) > (size_t)PANEL_SMEM_ROWS_BYTES) w >>= 1;
    if ((size_t)((b + CMAX - 1) / CMAX) * w * sizeof(cplx) > (size_t)PANEL_SMEM_ROWS_BYTES) return NEGF_EUNSUPPORTED;
    const size_t fixed = (2 * CMAX * PW + 2 * PW) * sizeof(cplx) + 2 * CMAX * sizeof(Cand);
    static bool attr_done = false;
    if (!attr_done) {
        NEGF_CUDA_CHECK(ctx, cudaFuncSetAttribute(gj_panel_cluster_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                  (int)(PANEL_SMEM_ROWS_BYTES + fixed)));
        NEGF_CUDA_CHECK(ctx, cudaFuncSetAttribute(gj_colperm_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
        NEGF_CUDA_CHECK(ctx, cudaFuncSetAttribute(gj_panel_reg_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(RegPanelSmem)));
        NEGF_CUDA_CHECK(ctx, cudaFuncSetAttribute(gj_panel_reg_kernel<256>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(RegPanelSmem)));
        attr_done = true;
    }
    const cplx one = cmake(1.0, 0.0), mone = cmake(-1.0, 0.0), zero = cmake(0.0, 0.0);
    // Two-level blocking.  Inside an outer block K = [K0, K0 + nbk) the width-w panels are
    // eliminated with their row swaps and rank-w updates restricted to the columns of K, so that
    // those columns end up holding Q = E[:, K] of the accumulated transform E (identity outside the
    // columns K); every other column then gets all nbk swaps at once and ONE rank-nbk update
    // M[:, ~K] = (M with rows K zeroed)[:, ~K] + Q R, R = the pivot rows: a GEMM with k = 128.
    for (int K0 = 0; K0 < b; K0 += OUTER_NB) {
      const int nbk = min(OUTER_NB, b - K0), K1 = K0 + nbk;
      for (int k0 = K0; k0 < K1; k0 += w) {
        const int wk = min(w, K1 - k0);
        const int rows = b - k0;
        const bool reg_panel = rows <= 2048;
        GemmArgs g;
        g.opA = 0; g.opB = 0; g.batch = batch; g.skip = skip;
        g.batch2 = 1; g.sA2 = g.sB2 = g.sD2 = g.sC2 = 0; g.alpha_vec = nullptr;
        cudaLaunchConfig_t cfg = {};
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.attrs = at; cfg.numAttrs = 1; cfg.stream = ctx->stream;
        if (reg_panel) {
            // one row per thread in registers; finishes P' (diagonal block and below) in place
            const int NT = rows <= 1024 ? 128 : 256;
            const int C = (rows + NT - 1) / NT;
            PanelArgs pa{A, sA, b, k0, wk, 0, W.ipiv, W.Dinv, W.Linv, info, info_code, skip};
            cfg.gridDim = dim3(C, batch); cfg.blockDim = dim3(NT); cfg.dynamicSmemBytes = sizeof(RegPanelSmem);
            at[0].val.clusterDim.x = C;
            if (NT == 128) NEGF_CUDA_CHECK(ctx, cudaLaunchKernelEx(&cfg, gj_panel_reg_kernel<128>, pa));
            else           NEGF_CUDA_CHECK(ctx, cudaLaunchKernelEx(&cfg, gj_panel_reg_kernel<256>, pa));
            ctx->launches++;
            if (nbk > wk) {
                gj_swap_extract_kernel<<<dim3((nbk + 127) / 128, batch), 128, 0, ctx->stream>>>(
                    A, sA, b, k0, wk, K0, K1, k0, k0 + wk, W.ipiv, W.R, skip);
                NEGF_LAUNCH_CHECK(ctx);
            }
            // rows above the panel: P' = -T Dinv, in place (each CTA reads exactly the rows it writes)
            if (k0 > 0) {
                g.alpha = mone; g.beta = zero; g.D = nullptr; g.sD = 0;
                g.m = k0; g.n = wk; g.k = wk; g.A = A + k0; g.lda = b; g.sA = sA;
                g.B = W.Dinv; g.ldb = wk; g.sB = PW * PW; g.C = A + k0; g.ldc = b; g.sC = sA;
                NEGF_TRY(zgemm_launch(ctx, g));
            }
            // M[:, other columns of K] += P' R, P' read from the panel's own columns
            g.alpha = one; g.beta = one; g.m = b; g.k = wk; g.A = A + k0; g.lda = b; g.sA = sA;
            g.ldb = b; g.sB = (long long)wk * b; g.ldc = b; g.sC = sA; g.sD = sA;
            if (k0 > K0) {
                g.n = k0 - K0; g.B = W.R + K0; g.C = A + K0; g.D = A + K0;
                NEGF_TRY(zgemm_launch(ctx, g));
            }
            if (k0 + wk < K1) {
                g.n = K1 - k0 - wk; g.B = W.R + k0 + wk; g.C = A + k0 + wk; g.D = A + k0 + wk;
                NEGF_TRY(zgemm_launch(ctx, g));
            }
            continue;
        }
        // cluster size: smallest power of two whose slabs fit, at least wk rows per slab
        // cluster size: smallest power of two whose slabs fit, at least wk rows per slab
        int C = 1;
        while (C < CMAX && (size_t)((rows + C - 1) / C) * wk * sizeof(cplx) > (size_t)PANEL_SMEM_ROWS_BYTES) C <<= 1;
        // more CTAs shorten the per-column elimination when the panel is tall
        while (C < CMAX && (rows + C - 1) / C > 512) C <<= 1;
        int slab = max(wk, (rows + C - 1) / C);
        PanelArgs pa{A, sA, b, k0, wk, slab, W.ipiv, W.Dinv, W.Linv, info, info_code, skip};
        cfg.gridDim = dim3(C, batch);
        cfg.blockDim = dim3(PANEL_NT);
        cfg.dynamicSmemBytes = (size_t)slab * wk * sizeof(cplx) + fixed;
        at[0].val.clusterDim.x = C;
        NEGF_CUDA_CHECK(ctx, cudaLaunchKernelEx(&cfg, gj_panel_cluster_kernel, pa));
        ctx->launches++;
        // row swaps on the other columns of K + pivot rows -> R, zeroed in A
        if (nbk > wk) {
            gj_swap_extract_kernel<<<dim3((nbk + 127) / 128, batch), 128, 0, ctx->stream>>>(
                A, sA, b, k0, wk, K0, K1, k0, k0 + wk, W.ipiv, W.R, skip);
            NEGF_LAUNCH_CHECK(ctx);
        }
        // P' = [-T Dinv ; Dinv ; -L21 Linv]
        g.alpha = mone; g.beta = zero; g.D = nullptr; g.sD = 0;
        g.n = wk; g.k = wk; g.ldb = wk; g.sB = PW * PW; g.ldc = wk; g.sC = (long long)b * wk; g.lda = b; g.sA = sA;
        if (k0 > 0) {
            g.m = k0; g.A = A + k0; g.B = W.Dinv; g.C = W.Pbuf;
            NEGF_TRY(zgemm_launch(ctx, g));
        }
        if (k0 + wk < b) {
            g.m = b - k0 - wk; g.A = A + (size_t)(k0 + wk) * b + k0; g.B = W.Linv; g.C = W.Pbuf + (size_t)(k0 + wk) * wk;
            NEGF_TRY(zgemm_launch(ctx, g));
        }
        gj_pbuf_diag_kernel<<<dim3((wk * wk + 255) / 256, batch), 256, 0, ctx->stream>>>(W.Pbuf, b, k0, wk, W.Dinv, skip);
        NEGF_LAUNCH_CHECK(ctx);
        // M[:, other columns of K] += P' R
        g.alpha = one; g.beta = one; g.m = b; g.k = wk; g.A = W.Pbuf; g.lda = wk; g.sA = (long long)b * wk;
        g.ldb = b; g.sB = (long long)wk * b; g.ldc = b; g.sC = sA; g.sD = sA;
        if (k0 > K0) {
            g.n = k0 - K0; g.B = W.R + K0; g.C = A + K0; g.D = A + K0;
            NEGF_TRY(zgemm_launch(ctx, g));
        }
        if (k0 + wk < K1) {
            g.n = K1 - k0 - wk; g.B = W.R + k0 + wk; g.C = A + k0 + wk; g.D = A + k0 + wk;
            NEGF_TRY(zgemm_launch(ctx, g));
        }
        gj_panel_store_kernel<<<dim3((b * wk + 255) / 256, batch), 256, 0, ctx->stream>>>(A, sA, b, k0, wk, W.Pbuf, W.Dinv, skip);
        NEGF_LAUNCH_CHECK(ctx);
      }
      if (nbk == b) break;       // a single outer block: nothing outside it
      // all nbk swaps of this outer block on the columns outside K; pivot rows -> Rout, zeroed in A
      gj_swap_extract_kernel<<<dim3((b + 127) / 128, batch), 128, 0, ctx->stream>>>(
          A, sA, b, K0, nbk, 0, b, K0, K1, W.ipiv, W.Rout, skip);
      NEGF_LAUNCH_CHECK(ctx);
      // M[:, ~K] += Q R with Q = M[:, K] in place
      GemmArgs g;
      g.opA = 0; g.opB = 0; g.alpha = one; g.beta = one; g.batch = batch; g.skip = skip;
      g.batch2 = 1; g.sA2 = g.sB2 = g.sD2 = g.sC2 = 0; g.alpha_vec = nullptr;
      g.m = b; g.k = nbk; g.A = A + K0; g.lda = b; g.sA = sA;
      g.ldb = b; g.sB = (long long)nbk * b; g.ldc = b; g.sC = sA; g.sD = sA;
      if (K0 > 0) {
          g.n = K0; g.B = W.Rout; g.C = A; g.D = A;
          NEGF_TRY(zgemm_launch(ctx, g));
      }
      if (K1 < b) {
          g.n = b - K1; g.B = W.Rout + K1; g.C = A + K1; g.D = A + K1;
          NEGF_TRY(zgemm_launch(ctx, g));
      }
    }
    gj_permidx_kernel<<<batch, 256, (size_t)b * sizeof(int), ctx->stream>>>(b, W.ipiv, W.idx, skip);
    NEGF_LAUNCH_CHECK(ctx);
    int rows_per = max(1, min(b, (4 * ctx->num_sms + batch - 1) / batch));
    gj_colperm_kernel<<<dim3(rows_per, batch), 256, (size_t)b * sizeof(cplx), ctx->stream>>>(A, sA, b, W.ipiv, W.idx, skip);
    NEGF_LAUNCH_CHECK(ctx);
    return NEGF_OK;
}

extern "C" int negf_zinverse_batched(negf_ctx* ctx, int b, negf_c128* A, long long stride, int batch, int* info) {
    if (!ctx || !A || b < 1 || batch < 0) return NEGF_EINVAL;
    size_t need = zinv_workspace_bytes(b, batch);
    if (b > SMALL_MAX && (!ctx->ws || ctx->ws_bytes < need)) return NEGF_ENOWORKSPACE;
    if (info) NEGF_CUDA_CHECK(ctx, cudaMemsetAsync(info, 0, sizeof(int) * batch, ctx->stream));
    return zinv_launch(ctx, b, (cplx*)A, stride, batch, ctx->ws, info, 0, nullptr);
}
