// K1: batched in-place complex inverse with partial pivoting.
//
// Every g_i = (A_ii - A_{i,i-1} g_{i-1} A_{i-1,i})^-1 of the RGF forward sweep (
// SURVEY.md 8(a) S3) and every g = a_b^-1 of the Sancho-Rubio doubling is one
// call of this file.
//
// Three regimes (zinv_launch at the end of the file picks one by block size):
//  * b <= 16 and 64 < b <= 96 (and every b <= 96 with NEGF_OPT_INV_TENSOR = 0): gj_reg_kernel - unblocked
//    Gauss-Jordan with the whole matrix in REGISTERS of one CTA of 16 warps, implicit threshold pivoting on a
//    32-bit key, one block barrier per column, look-ahead of the next column's pivot search;
//  * 16 < b <= 64: gj_dmma_kernel - blocked Gauss-Jordan in one CTA, panel width 4: one panel warp (alone on
//    its scheduler partition) factorises panel K+1 while 8 update warps apply panel K to the whole matrix as
//    a rank-4 update on the FP64 tensor pipe (DMMA.8x8x4), matrix in the accumulator layout + a shared copy;
//  * b > 96: two-level BLOCKED in-place Gauss-Jordan (outer blocks of 128 columns, panels of 32):
//      1. the panel is eliminated on ALL rows by gj_panel_rows_kernel (zinv_rows.cu: one matrix row per thread,
//         cluster of up to 8 CTAs, one block + one cluster barrier per column), which leaves the transform columns
//         P' = [-T D^-1 ; D^-1 ; -B D^-1] in place; blocks above 2048 rows (or NEGF_OPT_INV_PANEL = 0) use the first
//         generation instead: LU of the rows at and below the panel by gj_panel_reg_kernel (lane = panel column)
//         or gj_panel_cluster_kernel (panel in distributed shared memory), then P' from small GEMMs;
//      2. the panel's row swaps are applied to the other columns of the outer block, the pivot rows R are
//         moved to scratch and zeroed (gj_swap_extract_kernel);
//      3. rank-32 update of the other columns of the outer block: M += P' R (K2, DMMA);
//      4. after the 4 panels of an outer block: all 128 swaps on the columns outside it and ONE rank-128
//         update M[:, ~K] += Q R, Q = the block's own columns read in place (87 % of the flops at b = 1024);
//      5. the column permutation of the recorded swaps is undone at the end (gj_colperm_kernel).
//    Cost b^3 complex multiply-adds = 8 b^3 flops = 1 U, same as getrf + getri.  Pivoting is partial pivoting
//    among the not-yet-eliminated rows, exactly as in LU.
#include <cooperative_groups.h>

#include "common.cuh"
#include "zinv_rows.cuh"

namespace cg = cooperative_groups;

namespace {

constexpr int SMALL_MAX = 96;      // b*b*16 B <= 147 KB
constexpr int PW = 32;             // max panel width (one lane per panel column)
constexpr int CMAX = 8;            // portable cluster size
constexpr int PANEL_SMEM_ROWS_BYTES = 176 * 1024;   // + 9 KB exchange buffers + 33 KB static < 227 KB

// ------------------------------------------------------------------------------------------------
// small path: REGISTER-resident Gauss-Jordan, one CTA of 16 warps per matrix (b <= 96).
//   * warp w owns the columns j = w + 16 c (c < CB), lane l the rows i = l + 32 r (r < RB): the
//     whole matrix lives in registers (RB x CB elements per thread);
//   * the pivot search of column k is done by its owner warp alone with one redux.sync on a 32-bit
//     key made of the leading bits of |re|+|im| and the row, which then publishes the
//     multiplier column, the pivot index and 1/pivot to shared memory;
//   * ONE block barrier per column; the two rows that trade places travel inside each warp
//     through a per-warp shared-memory line (no block-level traffic);
//   * look-ahead: the owner of column k+1 updates that column first, searches its pivot and
//     publishes it BEFORE finishing its update for column k, so the barrier of column k+1 never
//     waits for a pivot search;
//   * the rank-1 update runs out of registers at the DFMA rate (= the DMMA rate on sm_100).
// Rows/columns >= b are padded with the identity and never reached.
// ------------------------------------------------------------------------------------------------


// 1 / a for a pivot (O(1): no overflow guard needed).  The real reciprocal is the hardware's 20-bit
// estimate refined by two Newton steps (2^-20 -> 2^-40 -> below one ulp): about 50 cycles of dependent
// latency instead of the ~80 of the IEEE division sequence, on the critical chain of every column.
__device__ __forceinline__ cplx crecip_fast(cplx a) {
    const double x = fma(a.x, a.x, a.y * a.y);
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    double e = fma(-x, r, 1.0);
    r = fma(r, e, r);
    e = fma(-x, r, 1.0);
    r = fma(r, e, r);
    return cmake(a.x * r, -a.y * r);
}

struct GjShared {            // pointers into the kernel's shared memory
    cplx* colbuf;            // [2][NR]
    cplx* wrow;              // this warp's [2][2][CB]
    cplx* s_d; int* s_p; int* piv; int* s_sing;
    cplx* rscale;            // [NR] pending scale 1/pivot of every row that has been a pivot row
};

// pivot search + publication of column kn, held in slot C of the calling (owner) warp
template <int RB, int CB, int C>
__device__ __forceinline__ void gj_owner(const cplx (&m)[RB][CB], unsigned used, const GjShared& sh, int kn, int b, int lane) {
    constexpr int NR = RB * 32;
    const int parn = kn & 1;
    // ONE 32-bit key per candidate: the top 25 bits of |re| + |im| (sign 0, exponent, 13 mantissa bits)
    // above 7 bits of 127 - row, so a single redux.sync.max names the pivot: the largest candidate up
    // to a relative 2^-13 (threshold pivoting; the growth bound changes by that factor), lowest row first
    // among those.  Rows here are < 96.
    unsigned key = 0u;
#pragma unroll
    for (int r = 0; r < RB; r++) {
        const int i = lane + 32 * r;
        sh.colbuf[parn * NR + i] = m[r][C];
        if (!((used >> r) & 1u) && i < b) {
            const unsigned hi = (unsigned)((unsigned long long)__double_as_longlong(cabs1(m[r][C])) >> 32);
            key = max(key, (hi & 0xffffff80u) | (unsigned)(127 - i));
        }
    }
    const unsigned kmax = __reduce_max_sync(0xffffffffu, key);
    const unsigned p = 127u - (kmax & 127u);
    const bool sing = (kmax >> 7) == 0u;           // every candidate is zero (or denormal)
    if (lane == (int)(p & 31u)) {        // the lane that holds the pivot inverts and publishes it
        cplx pv = m[0][C];
#pragma unroll
        for (int r = 1; r < RB; r++) if ((int)(p >> 5) == r) pv = m[r][C];
        sh.s_p[parn] = (int)p; sh.piv[kn] = (int)p;
        const cplx dn = sing ? cmake(1.0, 0.0) : crecip_fast(pv);
        sh.s_d[parn] = dn; sh.rscale[p] = dn;
        if (sing && *sh.s_sing == 0) *sh.s_sing = kn + 1;
    }
}

// Rank-1 update of column slot C: m[:, C] -= mult * sr.  The special rows/columns were prepared by
// the caller so that this one formula is right everywhere (pivot row: mult = 0, its scaling by 1/pivot
// stays pending; pivot column: m = 0 (1 in the pivot row), sr = 1/pivot -> -mult/pivot).
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

// all columns k = CK*NW + wk, wk < NW, then recurse to CK + 1
template <int RB, int CB, int GJ_NW, int CK>
__device__ __forceinline__ void gj_columns(cplx (&m)[RB][CB], unsigned& used, const GjShared& sh, int b, int warp, int lane) {
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
            cplx* wr = sh.wrow + par * CB;
            // IMPLICIT pivoting: rows never move.  The pivot row (physical row p) is broadcast inside
            // each warp through its shared-memory line and marked as used.  Its own scaling by 1/pivot
            // is DEFERRED (rscale[p], applied once in the final scatter): the registers keep the
            // unscaled row r_p, whose true value is d r_p.  Every later update of that row then needs
            // true_mult / d = the register value itself as multiplier, which is what the column
            // buffer holds, so pivoted and unpivoted rows run the same formula and the pivot row
            // costs no register traffic here (mult = 0 for this column).
            cplx mult[RB];
#pragma unroll
            for (int r = 0; r < RB; r++) {
                const int i = lane + 32 * r;
                mult[r] = sh.colbuf[par * NR + i];
                if (i == p) {
#pragma unroll
                    for (int c = 0; c < CB; c++) wr[c] = m[r][c];
                    mult[r] = cmake(0.0, 0.0);
                    used |= 1u << r;
                }
            }
            __syncwarp();
            cplx sr[CB];
#pragma unroll
            for (int c = 0; c < CB; c++) sr[c] = cmul(wr[c], d);
            if (warp == wk) {            // this warp's slot CK IS column k: -mult d, and 1 (= d / d) in the pivot row
                sr[CK] = d;
#pragma unroll
                for (int r = 0; r < RB; r++) m[r][CK] = cmake(lane + 32 * r == p ? 1.0 : 0.0, 0.0);
            }
            // look-ahead: the owner of column k+1 brings that column up to date and publishes it first
            int done = -1;
            if (k + 1 < b && warp == ((wk + 1) & (GJ_NW - 1))) {
                if (wk < GJ_NW - 1) {
                    gj_update<RB, CB, CK>(m, mult, sr);
                    gj_owner<RB, CB, CK>(m, used, sh, k + 1, b, lane);
                    done = CK;
                } else if (CK + 1 < CB) {
                    gj_update<RB, CB, CN>(m, mult, sr);
                    gj_owner<RB, CB, CN>(m, used, sh, k + 1, b, lane);
                    done = CN;
                }
            }
            gj_update_rest<RB, CB, 0>(m, mult, sr, done);
        }
        gj_columns<RB, CB, GJ_NW, CK + 1>(m, used, sh, b, warp, lane);
    }
}

template <int RB, int CB, int GJ_NW>
__global__ void __launch_bounds__(GJ_NW * 32) gj_reg_kernel(cplx* A, long long sA, int b, int* info, int code,
                                                            const int* skip, const int* code_dev) {
    constexpr int NR = RB * 32, NC = CB * GJ_NW;
    const int e = blockIdx.x;
    if (skip && skip[e]) return;
    __shared__ cplx colbuf[2 * NR];
    __shared__ cplx wrow[GJ_NW][2 * CB];         // [warp][parity][slot]: the pivot row of the current column
    __shared__ cplx s_d[2];
    __shared__ cplx rscale[NR];
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
    GjShared sh{colbuf, wrow[warp], s_d, s_p, piv, &s_sing, rscale};
    unsigned used = 0u;              // bit r: my row lane + 32 r has been a pivot row
    if (warp == 0) gj_owner<RB, CB, 0>(m, used, sh, 0, b, lane);
    gj_columns<RB, CB, GJ_NW, 0>(m, used, sh, b, warp, lane);
    __syncthreads();
    // With piv[k] = physical pivot row of column k the register array (times the pending row scales)
    // holds B[i][k] = X[i][piv[k]], X = Pi A^-1, Pi[piv[k]][k] = 1, so A^-1[r][piv[k]] = B[piv[r]][k]:
    // every thread scatters its elements to row pinv[i], column piv[j].
    if (tid < b) dest[piv[tid]] = tid;         // dest = pinv
    __syncthreads();
#pragma unroll
    for (int r = 0; r < RB; r++) {
        const int i = lane + 32 * r;
        const cplx rs = i < b ? rscale[i] : cmake(1.0, 0.0);
#pragma unroll
        for (int c = 0; c < CB; c++) {
            const int j = warp + GJ_NW * c;
            if (i < b && j < b) g[(size_t)dest[i] * b + piv[j]] = cmul(m[r][c], rs);
        }
    }
    if (tid == 0 && s_sing && info && info[e] == 0) info[e] = code_dev ? *code_dev + code : (code > 0 ? code : s_sing);   // first failure wins
}

// ------------------------------------------------------------------------------------------------
// small path, tensor-pipe variant: BLOCKED Gauss-Jordan inside one CTA (b <= 64), panel width 8.
//   * the matrix (padded with the identity to N = 32 TM) lives in the DMMA accumulator layout of
//     16 update warps (4 x 4 grid, warp tile 8 TM x 8 TM) AND as a copy in shared memory ("mirror",
//     double-buffered), which is where the panel columns and the pivot rows are read from;
//   * a 17th warp factorises the current 8-column panel on ALL N rows by in-place Gauss-Jordan with
//     partial pivoting among the not yet used rows (lane = row, the 8 columns in registers, straight-
//     line code: the pivot search + reciprocal of column j+1 are issued between the rank-1 updates of
//     column j).  The 8 stored columns are the transform T (N x 8) of the panel;
//   * all other columns then get ONE rank-8 update on the tensor pipe:
//         C <- C (pivot rows zeroed) + T R,   R[j, :] = row p_j of the matrix before the panel,
//     the panel columns themselves become T.  Two block barriers per panel instead of one per column.
// Rows never move (implicit pivoting); the permutation is undone in the final scatter, as above.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void gjd_dmma(double& c0, double& c1, double a, double b) {
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
        : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}
__device__ __forceinline__ double gjd_flip(double x) {
    return __hiloint2double(__double2hiint(x) ^ 0x80000000, __double2loint(x));
}

constexpr int GJD_UW = 8;                      // update warps (2 x 4 grid)
// 11 hardware warps (at most 3 per scheduler partition -> up to 168 registers per thread): warp 0 factorises
// the panels and has its scheduler partition to itself (warps 4 and 8 exit at once), because its dependent
// FP64 chain would otherwise queue behind the DMMAs of the update warps on the shared FP64 pipe; the update
// warps are the hardware warps 1-3, 5-7, 9-10.
constexpr int GJD_NT = 11 * 32;
constexpr int GJD_ACT = (GJD_UW + 1) * 32;     // threads that take part in the barriers
constexpr int GJD_W = 4;                       // panel width = one k-step of DMMA.8x8x4
template <int TM> constexpr size_t gjd_smem_bytes() {
    constexpr int N = 32 * TM, LD = N + 1, W = GJD_W;
    return (size_t)2 * N * LD * sizeof(cplx) + (size_t)4 * N * W * sizeof(cplx) + 16 * sizeof(cplx) + (4 * N + 16 + 4) * sizeof(int);
}

// pivot of panel column C (global column k): p = row (warp-uniform), d = 1 / pivot (computed by every lane)
template <int TM, int W, int C>
__device__ __forceinline__ void gjd_search(const cplx (&x)[TM][W], unsigned used, int k, int b, int lane, int& p, cplx& d, int& sing_at) {
    unsigned key = 0u;
#pragma unroll
    for (int r = 0; r < TM; r++) {
        const int i = lane + 32 * r;
        if (!((used >> r) & 1u) && ((i < b) == (k < b))) {
            const unsigned hi = (unsigned)((unsigned long long)__double_as_longlong(cabs1(x[r][C])) >> 32);
            key = max(key, (hi & 0xffffff80u) | (unsigned)(127 - i));
        }
    }
    const unsigned kmax = __reduce_max_sync(0xffffffffu, key);
    p = 127 - (int)(kmax & 127u);
    const bool sing = (kmax >> 7) == 0u;
    double vx = x[0][C].x, vy = x[0][C].y;
#pragma unroll
    for (int r = 1; r < TM; r++) if ((p >> 5) == r) { vx = x[r][C].x; vy = x[r][C].y; }
    vx = __shfl_sync(0xffffffffu, vx, p & 31);
    vy = __shfl_sync(0xffffffffu, vy, p & 31);
    d = sing ? cmake(1.0, 0.0) : crecip_fast(cmake(vx, vy));
    sing_at = (sing && sing_at == 0) ? k + 1 : sing_at;
}

// one Gauss-Jordan step of the panel (column J) + look-ahead search of column J+1.
// Tt receives the coefficients AS APPLIED: row i gets  row_i += Tt[i][J] x (pivot row p_J as it is at step J),
// Tt[p_J][J] = 1 / pivot (the pivot row is replaced by its scaled self); pjx[p_J] = J + 1.
template <int TM, int W, int J>
__device__ __forceinline__ void gjd_panel_steps(cplx (&x)[TM][W], cplx (&rsc)[TM], unsigned& used,
                                                int& p, cplx& d, int& myp, int& sing_at, int k0, int b, int lane,
                                                cplx* prow_s, cplx* Tt, int* pjx) {
    if constexpr (J < W) {
        const int pl = p & 31, pr = p >> 5;
        cplx* line = prow_s + (J & 1) * 8;
#pragma unroll
        for (int r = 0; r < TM; r++)
            if (lane == pl && pr == r) {
#pragma unroll
                for (int c = 0; c < W; c++) line[c] = x[r][c];
                pjx[p] = J + 1;
            }
        myp = (lane == J) ? p : myp;
        __syncwarp();
        // deferred scaling inside the panel: the registers of a pivot row keep the unscaled row (true value =
        // rsc x register), so pivoted and unpivoted rows run the same update and the pivot row itself costs nothing
        cplx mlt[TM];
#pragma unroll
        for (int r = 0; r < TM; r++) {
            const bool isp = (lane == pl) && (pr == r);
            const cplx t = cmul(x[r][J], d);
            mlt[r] = isp ? cmake(0.0, 0.0) : t;
            x[r][J] = isp ? cmake(1.0, 0.0) : cneg(t);
            const cplx tt = cmul(t, rsc[r]);                   // true coefficient of a row pivoted earlier in this panel
            Tt[(lane + 32 * r) * W + J] = isp ? d : cneg(tt);
            if (isp) { rsc[r] = d; used |= 1u << r; }
        }
        int pn = 0; cplx dn = cmake(1.0, 0.0);
        if constexpr (J < W - 1) {
            const cplx prn = line[J + 1];
#pragma unroll
            for (int r = 0; r < TM; r++) cfms(x[r][J + 1], mlt[r], prn);
            gjd_search<TM, W, J + 1>(x, used, k0 + J + 1, b, lane, pn, dn, sing_at);
        }
#pragma unroll
        for (int c = 0; c < W; c++) {
            if (c == J || c == J + 1) continue;
            const cplx prc = line[c];
#pragma unroll
            for (int r = 0; r < TM; r++) cfms(x[r][c], mlt[r], prc);
        }
        p = pn; d = dn;
        gjd_panel_steps<TM, W, J + 1>(x, rsc, used, p, d, myp, sing_at, k0, b, lane, prow_s, Tt, pjx);
    }
}

__device__ __forceinline__ void gjd_bar_sync(int id, int count) { asm volatile("bar.sync %0, %1;" :: "r"(id), "r"(count) : "memory"); }
__device__ __forceinline__ void gjd_bar_arrive(int id, int count) { __threadfence_block(); asm volatile("bar.arrive %0, %1;" :: "r"(id), "r"(count) : "memory"); }

// B operand of the rank-4 update for matrix column `col` (lane = (g: column, q: pivot index)): the pivot row
// p_q AS IT IS WHEN IT IS USED, i.e. after the steps l < q of this panel have been applied to it:
//   R~_q = R_q + sum_{l<q} Tt[p_q][l] R~_l      (lanes q = l are final after l rounds).
// With this operand and the as-applied coefficients as A operand the DMMA accumulates, per element and in
// the same order, exactly the updates of the unblocked elimination (bounded multipliers); the product
// form T R with the original rows would go through the explicit inverse of the 4 x 4 pivot block instead.
__device__ __forceinline__ cplx gjd_bfrag(const cplx* mc, int LD, const cplx* Tt, int pq, int col, int q, int lane) {
    cplx v = mc[pq * LD + col];
#pragma unroll
    for (int l = 0; l < GJD_W - 1; l++) {
        const int src = (lane & ~3) + l;
        const double sx = __shfl_sync(0xffffffffu, v.x, src), sy = __shfl_sync(0xffffffffu, v.y, src);
        if (q > l) cfma(v, Tt[pq * GJD_W + l], cmake(sx, sy));
    }
    return v;
}

// Look-ahead: while the update warps apply panel K to the matrix, the panel warp already factorises
// panel K+1.  For that the update warps FIRST bring the columns of panel K+1 up to date (one 8 x 8 row
// tile per warp, accumulator taken from and written back to the mirror), signal the panel warp
// (named barrier A) and only then update their own tiles (which repeats that tile bit for bit).
// Named barriers: 1 = update warps only (mirror complete), 2/3 = panel K factorised (panel warp
// arrives, update warps wait), 4/5 = columns of panel K ready in the mirror (update warps arrive,
// panel warp waits).  The panel outputs are double-buffered.
template <int TM>
__global__ void __launch_bounds__(GJD_NT, 1) gj_dmma_kernel(cplx* A, long long sA, int b, int* info, int code,
                                                            const int* skip, const int* code_dev) {
    // N = 32 TM rows; update warps in a 2 x 4 grid, warp tile (8 TR) x (8 TC) = TR x TC accumulator tiles
    constexpr int N = 32 * TM, LD = N + 1, TR = 2 * TM, TC = TM, WC = 4, NRT = N / 8, UT = GJD_UW * 32, W = GJD_W;
    constexpr int PPT = 8 / W;                   // panels per 8-column tile
    const int e = blockIdx.x;
    pdl_wait();                                  // programmatic dependent launch (common.cuh)
    pdl_trigger();
    if (skip && skip[e]) return;
    extern __shared__ __align__(16) unsigned char gjd_smem[];
    cplx* mir = (cplx*)gjd_smem;                 // [2][N][LD]
    cplx* Tb = mir + 2 * N * LD;                 // [2][N][W]  final panel columns (the transform T)
    cplx* Ttb = Tb + 2 * N * W;                  // [2][N][W]  coefficients as applied
    cplx* prow_s = Ttb + 2 * N * W;              // [2][8]
    int* piv = (int*)(prow_s + 16);              // [N]
    int* dest = piv + N;                         // [N]
    int* pjxb = dest + N;                        // [2][N]  j + 1 for the j-th pivot row of the panel, else 0
    int* prows = pjxb + 2 * N;                   // [2][8]
    int* s_sing = prows + 16;
    const int hw = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (hw == 4 || hw == 8) return;
    const int warp = hw == 0 ? GJD_UW : hw - 1 - (hw > 4) - (hw > 8);    // 0..7 update warps, 8 = panel warp
    const int tid = warp * 32 + lane;
    const int g = lane >> 2, q = lane & 3, wr = (warp >> 2) & 1, wc = warp & 3;
    const int row0 = 8 * TR * wr + g, col0 = 8 * TC * wc + 2 * q;     // + 8 tr, + 8 tc (+ h)
    cplx* gA = A + (size_t)e * sA;
    const int npanel = (b + W - 1) / W;
    double cre[TR][TC][2], cim[TR][TC][2];       // update warps: my accumulator tiles
    if (warp < GJD_UW) {
#pragma unroll
        for (int tr = 0; tr < TR; tr++)
#pragma unroll
            for (int tc = 0; tc < TC; tc++)
#pragma unroll
                for (int h = 0; h < 2; h++) {
                    const int i = row0 + 8 * tr, j = col0 + 8 * tc + h;
                    const cplx v = (i < b && j < b) ? gA[(size_t)i * b + j] : cmake(i == j ? 1.0 : 0.0, 0.0);
                    cre[tr][tc][h] = v.x; cim[tr][tc][h] = v.y;
                    mir[i * LD + j] = v;
                }
    }
    if (tid == 0) *s_sing = 0;
    gjd_bar_sync(0, GJD_ACT);
    if (warp == GJD_UW) {
        // ---------------- panel warp ----------------
        unsigned used = 0u;                      // bit r = my row lane + 32 r has been a pivot row
        int sing_at = 0;
#pragma unroll 1
        for (int K = 0; K < npanel; K++) {
            if (K > 0) gjd_bar_sync(4 + (K & 1), GJD_ACT);
            const cplx* mc = mir + (K & 1) * N * LD;
            int* pjx = pjxb + (K & 1) * N;
            cplx x[TM][W], rsc[TM];
#pragma unroll
            for (int r = 0; r < TM; r++) {
                rsc[r] = cmake(1.0, 0.0);
                pjx[lane + 32 * r] = 0;
#pragma unroll
                for (int c = 0; c < W; c++) x[r][c] = mc[(lane + 32 * r) * LD + W * K + c];
            }
            __syncwarp();
            int p, myp = 0; cplx d;
            gjd_search<TM, W, 0>(x, used, W * K, b, lane, p, d, sing_at);
            gjd_panel_steps<TM, W, 0>(x, rsc, used, p, d, myp, sing_at, W * K, b, lane, prow_s, Ttb + (K & 1) * N * W, pjx);
            cplx* Tk = Tb + (K & 1) * N * W;
#pragma unroll
            for (int r = 0; r < TM; r++)
#pragma unroll
                for (int c = 0; c < W; c++) Tk[(lane + 32 * r) * W + c] = cmul(x[r][c], rsc[r]);
            if (lane < W) { piv[W * K + lane] = myp; prows[(K & 1) * 8 + lane] = myp; }
            gjd_bar_arrive(2 + (K & 1), GJD_ACT);
        }
        if (lane == 0 && sing_at) *s_sing = sing_at;
    } else {
        // ---------------- update warps ----------------
#pragma unroll 1
        for (int Kc = 0; Kc < WC; Kc++) {
#pragma unroll
            for (int tcs = 0; tcs < TC; tcs++) {
#pragma unroll
                for (int hp = 0; hp < PPT; hp++) {
                    const int K = (Kc * TC + tcs) * PPT + hp;
                    if (K >= npanel) break;
                    const bool more = K + 1 < npanel;
                    const cplx* mc = mir + (K & 1) * N * LD;
                    cplx* mn = mir + ((K + 1) & 1) * N * LD;
                    const cplx* Tk = Tb + (K & 1) * N * W;
                    const cplx* Tt = Ttb + (K & 1) * N * W;
                    const int* pjx = pjxb + (K & 1) * N;
                    gjd_bar_sync(2 + (K & 1), GJD_ACT);
                    const int pq = prows[(K & 1) * 8 + q];
                    if (more) {
                        // early tile: rows 8 warp .. + 7 of the 8-column tile that holds panel K+1 (all warps run the
                        // shuffles of the operand; the warps beyond the last row tile only skip the product)
                        const int cb = ((K + 1) / PPT) * 8;
                        const cplx tb = gjd_bfrag(mc, LD, Tt, pq, cb + g, q, lane);
                        if (warp < NRT) {
                            const int i = 8 * warp + g, j = cb + 2 * q;
                            const int pj = pjx[i];
                            cplx c0 = mc[i * LD + j], c1 = mc[i * LD + j + 1];
                            if (pj) { c0 = cmake(0.0, 0.0); c1 = c0; }
                            cplx ta = Tt[i * W + q];
                            if (q < pj - 1) ta = cmake(0.0, 0.0);
                            gjd_dmma(c0.x, c1.x, ta.x, tb.x);
                            gjd_dmma(c0.y, c1.y, ta.x, tb.y);
                            gjd_dmma(c0.x, c1.x, ta.y, gjd_flip(tb.y));
                            gjd_dmma(c0.y, c1.y, ta.y, tb.x);
                            if ((q >> 1) == ((K + 1) & 1)) { mn[i * LD + j] = c0; mn[i * LD + j + 1] = c1; }
                        }
                        gjd_bar_arrive(4 + ((K + 1) & 1), GJD_ACT);
                    }
                    double are[TR], aim[TR], bre[TC], bim[TC], bni[TC];
#pragma unroll
                    for (int t = 0; t < TC; t++) {
                        const cplx tb = gjd_bfrag(mc, LD, Tt, pq, 8 * TC * wc + 8 * t + g, q, lane);
                        bre[t] = tb.x; bim[t] = tb.y; bni[t] = gjd_flip(tb.y);
                    }
#pragma unroll
                    for (int tr = 0; tr < TR; tr++) {
                        const int i = row0 + 8 * tr;
                        const int pj = pjx[i];
                        cplx ta = Tt[i * W + q];
                        if (q < pj - 1) ta = cmake(0.0, 0.0);      // the steps before a pivot row's own are inside R~
                        are[tr] = ta.x; aim[tr] = ta.y;
                        if (pj) {
#pragma unroll
                            for (int tc = 0; tc < TC; tc++) { cre[tr][tc][0] = cre[tr][tc][1] = 0.0; cim[tr][tc][0] = cim[tr][tc][1] = 0.0; }
                        }
                    }
#pragma unroll
                    for (int tc = 0; tc < TC; tc++) {
#pragma unroll
                        for (int tr = 0; tr < TR; tr++) {
                            gjd_dmma(cre[tr][tc][0], cre[tr][tc][1], are[tr], bre[tc]);
                            gjd_dmma(cim[tr][tc][0], cim[tr][tc][1], are[tr], bim[tc]);
                            gjd_dmma(cre[tr][tc][0], cre[tr][tc][1], aim[tr], bni[tc]);
                            gjd_dmma(cim[tr][tc][0], cim[tr][tc][1], aim[tr], bre[tc]);
                        }
                        // my columns of panel K itself become T
                        if (tc == tcs && wc == Kc && (q >> 1) == hp) {
#pragma unroll
                            for (int tr = 0; tr < TR; tr++)
#pragma unroll
                                for (int h = 0; h < 2; h++) {
                                    const cplx t = Tk[(row0 + 8 * tr) * W + ((2 * q + h) & (W - 1))];
                                    cre[tr][tc][h] = t.x; cim[tr][tc][h] = t.y;
                                }
                        }
#pragma unroll
                        for (int tr = 0; tr < TR; tr++)
#pragma unroll
                            for (int h = 0; h < 2; h++)
                                mn[(row0 + 8 * tr) * LD + col0 + 8 * tc + h] = cmake(cre[tr][tc][h], cim[tr][tc][h]);
                    }
                    gjd_bar_sync(1, UT);
                }
            }
        }
        // as in gj_reg_kernel: the accumulators hold B[i][k] = X[i][piv[k]], X = Pi A^-1, so
        // A^-1[pinv[i]][piv[j]] = B[i][j]; dest = pinv
        if (tid < b) dest[piv[tid]] = tid;
        gjd_bar_sync(1, UT);
#pragma unroll
        for (int tr = 0; tr < TR; tr++) {
            const int i = row0 + 8 * tr;
            if (i >= b) continue;
            cplx* orow = gA + (size_t)dest[i] * b;
#pragma unroll
            for (int tc = 0; tc < TC; tc++)
#pragma unroll
                for (int h = 0; h < 2; h++) {
                    const int j = col0 + 8 * tc + h;
                    if (j < b) orow[piv[j]] = cmake(cre[tr][tc][h], cim[tr][tc][h]);
                }
        }
    }
    gjd_bar_sync(0, GJD_ACT);                    // the panel warp's singular flag
    if (tid == 0 && *s_sing && info && info[e] == 0) info[e] = code_dev ? *code_dev + code : (code > 0 ? code : *s_sing);
}

// ------------------------------------------------------------------------------------------------
// blocked path, step 1: cluster panel LU with partial pivoting
// ------------------------------------------------------------------------------------------------
struct Cand { double val; int row; int pad; };
constexpr size_t PANEL_SMEM_FIXED = (2 * CMAX * PW + 2 * PW) * sizeof(cplx) + 2 * CMAX * sizeof(Cand);

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
// step 1, register-resident variant (tall panels up to 8 x 256 rows).  Lane = panel column, every
// warp keeps R consecutive rows of the width-32 panel in registers (one complex per lane and row),
// 16 warps per CTA, a cluster of C CTAs covers the rows >= k0.  Per column: each warp's lane j
// scans its R rows, redux picks the CTA candidate, ONE DSMEM exchange (candidate key, row index,
// row content, current diagonal row) and ONE cluster barrier; the elimination is a shuffle
// broadcast of the multiplier plus one complex FMA per row, out of registers.  The kernel also
// finishes the panel in place: rows below the diagonal block leave as -L21 L11^-1, the diagonal
// block as (L11 U11)^-1, so the trailing GEMM reads P' straight from A's columns.
// (A first version with one ROW per thread needed ~1850 instructions per column and warp - the
// column index had to be picked by predication - and was instruction-latency bound; this layout
// needs ~300, see profiles/r01b_inverse.md.)
// ------------------------------------------------------------------------------------------------
constexpr int PNL_WARPS = 16;
constexpr int PNL_NONE = 0x7fffffff;

struct RegPanelSmem {
    cplx candrow[2][CMAX][PW];
    cplx diagrow[2][PW];
    cplx wrows[PNL_WARPS][PW];   // every warp's candidate row of the current column
    cplx drowstage[PW];
    cplx Dm[PW * PW];      // factored diagonal block L11 \ U11
    cplx Li[PW * PW];      // L11^-1 (every CTA gets a copy)
    cplx Ui[PW * PW];      // U11^-1 (CTA 0)
    unsigned long long red_key[PNL_WARPS];
    int red_row[PNL_WARPS];
    unsigned long long cand_key[2][CMAX];
    int cand_row[2][CMAX];
    cplx Lrow[1];          // [PNL_WARPS * R][PW] follows (dynamic)
};

// argmax of (key, smallest row) over the lanes that hold a candidate; every lane gets the result
__device__ __forceinline__ void warp_best(unsigned long long key, int row, unsigned long long& bk, int& br) {
    const bool has = row != PNL_NONE;
    const unsigned hi = __reduce_max_sync(0xffffffffu, has ? (unsigned)(key >> 32) : 0u);
    const bool mh = has && (unsigned)(key >> 32) == hi;
    const unsigned lo = __reduce_max_sync(0xffffffffu, mh ? (unsigned)key : 0u);
    const bool ml = mh && (unsigned)key == lo;
    br = (int)__reduce_min_sync(0xffffffffu, ml ? (unsigned)row : (unsigned)PNL_NONE);
    bk = ((unsigned long long)hi << 32) | lo;
}

inline size_t reg_panel_smem_bytes(int R) { return sizeof(RegPanelSmem) + (size_t)PNL_WARPS * R * PW * sizeof(cplx); }

// Triangular inverses of the factored w x w diagonal block S.Dm = L11 \\ U11 by one warp each, lane = column c,
// the column held in registers: row r of the result needs rows k < r (k > r) of the same column, so the sums run
// over registers and broadcast reads of the factor, fully unrolled (the entries outside the triangles come out
// as exact zeros).  S.Li / S.Ui are zero-initialised by the caller.
__device__ __noinline__ void panel_tri_lower(RegPanelSmem& S, int w, int lane) {     // L11^-1 (unit lower)
    constexpr int H = PW / 2;
    // rows 0 .. 15 of column `lane` in registers; then rows 16 .. 31, which read the first half back from
    // shared memory (16 registers of column at a time keep the whole thing inside the register budget)
    {
        cplx li[H];
#pragma unroll
        for (int r = 0; r < H; r++) {
            li[r] = cmake(0.0, 0.0);
            if (r < w) {
                cplx s0 = cmake(r == lane ? 1.0 : 0.0, 0.0), s1 = cmake(0.0, 0.0);
#pragma unroll
                for (int k = 0; k < r; k++) {
                    if (k & 1) cfms(s1, S.Dm[r * PW + k], li[k]); else cfms(s0, S.Dm[r * PW + k], li[k]);
                }
                li[r] = cadd(s0, s1);
                S.Li[r * PW + lane] = li[r];
            }
        }
    }
    __syncwarp();
    cplx lj[H];
#pragma unroll
    for (int r = H; r < PW; r++) {
        lj[r - H] = cmake(0.0, 0.0);
        if (r < w) {
            cplx s0 = cmake(r == lane ? 1.0 : 0.0, 0.0), s1 = cmake(0.0, 0.0);
#pragma unroll
            for (int k = 0; k < H; k++) {
                if (k & 1) cfms(s1, S.Dm[r * PW + k], S.Li[k * PW + lane]); else cfms(s0, S.Dm[r * PW + k], S.Li[k * PW + lane]);
            }
#pragma unroll
            for (int k = H; k < r; k++) {
                if (k & 1) cfms(s1, S.Dm[r * PW + k], lj[k - H]); else cfms(s0, S.Dm[r * PW + k], lj[k - H]);
            }
            lj[r - H] = cadd(s0, s1);
            S.Li[r * PW + lane] = lj[r - H];
        }
    }
}
__device__ __noinline__ void panel_tri_upper(RegPanelSmem& S, int w, int lane) {     // U11^-1
    constexpr int H = PW / 2;
    {
        const cplx ur = S.Dm[lane * PW + lane];
        S.drowstage[lane] = (lane >= w || (ur.x == 0.0 && ur.y == 0.0)) ? cmake(0.0, 0.0) : crecip(ur);
    }
    __syncwarp();
    // rows 31 .. 16 first (registers), then rows 15 .. 0 with the upper half read back from shared memory;
    // Dm[r][k] = 0 for k >= w and Ui is zero-initialised, so the fixed ranges are right for w < 32 too
    {
        cplx ui[H];
#pragma unroll
        for (int r = PW - 1; r >= H; r--) {
            ui[r - H] = cmake(0.0, 0.0);
            if (r < w) {
                cplx s0 = cmake(r == lane ? 1.0 : 0.0, 0.0), s1 = cmake(0.0, 0.0);
#pragma unroll
                for (int k = r + 1; k < PW; k++) {
                    if (k & 1) cfms(s1, S.Dm[r * PW + k], ui[k - H]); else cfms(s0, S.Dm[r * PW + k], ui[k - H]);
                }
                ui[r - H] = cmul(cadd(s0, s1), S.drowstage[r]);
                S.Ui[r * PW + lane] = ui[r - H];
            }
        }
    }
    __syncwarp();
    cplx uj[H];
#pragma unroll
    for (int r = H - 1; r >= 0; r--) {
        uj[r] = cmake(0.0, 0.0);
        if (r < w) {
            cplx s0 = cmake(r == lane ? 1.0 : 0.0, 0.0), s1 = cmake(0.0, 0.0);
#pragma unroll
            for (int k = H; k < PW; k++) {
                if (k & 1) cfms(s1, S.Dm[r * PW + k], S.Ui[k * PW + lane]); else cfms(s0, S.Dm[r * PW + k], S.Ui[k * PW + lane]);
            }
#pragma unroll
            for (int k = r + 1; k < H; k++) {
                if (k & 1) cfms(s1, S.Dm[r * PW + k], uj[k]); else cfms(s0, S.Dm[r * PW + k], uj[k]);
            }
            uj[r] = cmul(cadd(s0, s1), S.drowstage[r]);
            S.Ui[r * PW + lane] = uj[r];
        }
    }
}

template <int R>
__global__ void __launch_bounds__(PNL_WARPS * 32) gj_panel_reg_kernel(PanelArgs a) {
    constexpr int NT = PNL_WARPS * 32;
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
    const int row0 = (rank * PNL_WARPS + warp) * R;               // first candidate row of this warp
    cplx* g = a.A + (size_t)e * a.sA + (size_t)k0 * b + k0;       // panel origin
    cplx P[R];
#pragma unroll
    for (int r = 0; r < R; r++)
        P[r] = (row0 + r < rows_total && lane < w) ? g[(size_t)(row0 + r) * b + lane] : cmake(0.0, 0.0);

#pragma unroll 1
    for (int j = 0; j < w; j++) {
        const int par = j & 1;
        // lane j scans its column over this warp's rows with index >= j (all lanes run the same code)
        unsigned long long key = 0ull; int row = PNL_NONE;
#pragma unroll
        for (int r = 0; r < R; r++) {
            const int gr = row0 + r;
            if (gr >= j && gr < rows_total) {
                const unsigned long long kq = (unsigned long long)__double_as_longlong(cabs1(P[r]));
                if (row == PNL_NONE || kq > key) { key = kq; row = gr; }
            }
        }
        key = __shfl_sync(0xffffffffu, key, j);
        row = __shfl_sync(0xffffffffu, row, j);
        {   // this warp's candidate row (and the current diagonal row, if it lives here) go to shared memory
            cplx v = cmake(0.0, 0.0);
#pragma unroll
            for (int r = 0; r < R; r++)
                if (row0 + r == row) v = P[r];
            S.wrows[warp][lane] = v;
            if (j >= row0 && j < row0 + R) {           // warp-uniform: only the warp that holds row j
                cplx dv = cmake(0.0, 0.0);
#pragma unroll
                for (int r = 0; r < R; r++)
                    if (row0 + r == j) dv = P[r];
                S.drowstage[lane] = dv;
            }
            if (lane == 0) { S.red_key[warp] = key; S.red_row[warp] = row; }
        }
        __syncthreads();
        if (warp == 0) {       // CTA candidate; push (key, row, row content) to every CTA; CTA 0 also the diagonal row
            // lane q holds warp q's candidate; argmax by three redux.sync (ties: the smallest row, as rows ascend with q)
            unsigned long long bk = 0ull; int br = PNL_NONE;
            warp_best(lane < PNL_WARPS ? S.red_key[lane] : 0ull, lane < PNL_WARPS ? S.red_row[lane] : PNL_NONE, bk, br);
            const int bw = br == PNL_NONE ? 0 : br / R - rank * PNL_WARPS;
            const cplx myrow = S.wrows[bw][lane];
            const cplx drow = S.drowstage[lane];
            if (C == 1) {
                S.candrow[par][0][lane] = myrow; S.diagrow[par][lane] = drow;
                if (lane == 0) { S.cand_key[par][0] = bk; S.cand_row[par][0] = br; }
            } else {
                for (int q = 0; q < C; q++) {
                    RegPanelSmem* Rm = cluster.map_shared_rank(&S, q);
                    Rm->candrow[par][rank][lane] = myrow;
                    if (rank == 0) Rm->diagrow[par][lane] = drow;
                    if (lane == 0) { Rm->cand_key[par][rank] = bk; Rm->cand_row[par][rank] = br; }
                }
            }
        }
        if (C == 1) __syncthreads(); else cluster.sync();
        // everybody picks the same winner; rows are contiguous per CTA, so the row names its CTA
        unsigned long long wk = 0ull; int prow = PNL_NONE;
        for (int q = 0; q < C; q++) {
            const unsigned long long k2 = S.cand_key[par][q]; const int r2 = S.cand_row[par][q];
            if (r2 != PNL_NONE && (prow == PNL_NONE || k2 > wk)) { wk = k2; prow = r2; }             // rows ascend with q
        }
        const bool sing = (prow == PNL_NONE) || wk == 0ull;
        if (prow == PNL_NONE) prow = j;
        const int wq = min(prow / (PNL_WARPS * R), C - 1);
        if (rank == 0 && tid == 0) {
            a.ipiv[(size_t)e * b + k0 + j] = k0 + prow;
            if (sing && a.info && a.info[e] == 0) a.info[e] = a.code > 0 ? a.code : (k0 + j + 1);
        }
        const cplx prl = sing ? cmake(0.0, 0.0) : S.candrow[par][wq][lane];
        const cplx pjv = S.candrow[par][wq][j];
        const cplx rinv = sing ? cmake(0.0, 0.0) : crecip_fast(pjv);
        const cplx dgl = S.diagrow[par][lane];
        // exchange rows j <-> prow: warp-uniform, only the (at most two) warps that hold one of them
        if (prow != j && ((prow >= row0 && prow < row0 + R) || (j >= row0 && j < row0 + R))) {
#pragma unroll
            for (int r = 0; r < R; r++) {
                const int gr = row0 + r;
                if (gr == prow) P[r] = dgl;
                else if (gr == j) P[r] = prl;
            }
        }
#pragma unroll
        for (int r = 0; r < R; r++) {
            const int gr = row0 + r;
            if (gr > j && gr < rows_total) {                       // eliminate below (warp-uniform test)
                cplx pj;
                pj.x = __shfl_sync(0xffffffffu, P[r].x, j);
                pj.y = __shfl_sync(0xffffffffu, P[r].y, j);
                const cplx l = cmul(pj, rinv);
                if (lane == j) P[r] = l;
                else if (lane > j) cfms(P[r], l, prl);
            }
        }
    }

    // every warp parks its rows in its own shared-memory lines now (read back for P' below), so that the
    // panel registers are free during the triangular inverses
    cplx* Lr = S.Lrow + (size_t)warp * R * PW;
#pragma unroll
    for (int r = 0; r < R; r++) Lr[r * PW + lane] = P[r];
    __syncwarp();
    // CTA 0: L11^-1 and U11^-1 from the w x w diagonal block, one warp each; then
    // (L11 U11)^-1 = U11^-1 L11^-1; L11^-1 goes to every CTA of the cluster.
    if (rank == 0) {
        for (int idx = tid; idx < PW * PW; idx += NT) { S.Li[idx] = cmake(0.0, 0.0); S.Ui[idx] = cmake(0.0, 0.0); }
#pragma unroll
        for (int r = 0; r < R; r++)
            if (row0 + r < PW) S.Dm[(row0 + r) * PW + lane] = Lr[r * PW + lane];
        __syncthreads();
        // triangular inverses by two warps (own functions, so that their register arrays do not weigh on the
        // column loop's allocation)
        if (warp == 0) panel_tri_lower(S, w, lane);
        else if (warp == 1) panel_tri_upper(S, w, lane);
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
    // rows below the diagonal block: P' = -L21 L11^-1, written in place (lane = output column)
#pragma unroll 1
    for (int r = 0; r < R; r++) {
        const int gr = row0 + r;
        if (gr >= w && gr < rows_total) {
            cplx acc = cmake(0.0, 0.0);
#pragma unroll 8
            for (int k = 0; k < PW; k++) cfms(acc, Lr[r * PW + k], S.Li[k * PW + lane]);   // Li[k][c] = 0 for k < c, k >= w
            if (lane < w) g[(size_t)gr * b + lane] = acc;
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

constexpr int OUTER_NB_MAX = 256;  // widest outer block of the two-level blocked Gauss-Jordan (sizes the scratch)
// Outer block width: the rank-nb update of all other columns is a GEMM with k = nb, the rank-32 updates inside
// the block grow with nb, and the look-ahead has more (shorter) stages with a small nb.  Measured (kernel_bench
// --kernel zinv, ms per batched inverse, nb = 64 / 128 / 256): b = 256 batch 256: 3.19 / 3.29 / 3.89; b = 512
// batch 32: 3.14 / 3.00 / 3.38; b = 1024 batch 8: 5.13 / 5.38 / 5.77; b = 2048 batch 8: 33.6 / 28.4 / 27.5.
// NEGF_OPT_INV_OUTER overrides (multiple of 32, <= 256).
// With the addend prefetch of K2 (zgemm.cu) re-measured, nb = 64 / 128 / 256: b = 256 batch 256: 2.92 / 3.02 / 3.37; b = 512
// batch 32: 2.91 / 2.91 / 3.26; b = 1024 batch 8: 4.76 / 5.18 / 5.71, batch 32: 15.36 / 14.33 / 14.73 (a large batch fills the
// machine without the look-ahead's many short stages); b = 2048 batch 8: 29.3 / 26.5 / 26.4.
// Last build of round 2 (K2's two-CTA tiles, merged rank-32 updates), nb = 64 / 128 / 256: b = 256 batch 256: 2.60 / 2.63 / 2.83;
// b = 512 batch 32: 2.71 / 2.65 / 2.81; b = 1024 batch 8: 4.45 / 5.03 / 5.13, batch 32: 13.30 / 12.65 / 12.78; b = 2048 batch 8:
// 25.8 / 24.1 / 23.6: the table below still picks the best of each row.
inline int outer_nb(const negf_ctx* ctx, int b, int batch) {
    if (ctx->inv_outer >= 32 && ctx->inv_outer <= OUTER_NB_MAX && ctx->inv_outer % 32 == 0) return ctx->inv_outer;
    if (b > 1024) return 256;
    if (b > 512) return batch >= 16 ? 128 : 64;
    return b > 256 ? 128 : 64;
}

struct InvWs {
    cplx* Rout;   // [batch][OUTER_NB_MAX][b]  pivot rows of an outer block
    cplx* R;      // [batch][PW][b]
    cplx* Pbuf;   // [batch][b][PW]
    cplx* Dinv;   // [batch][PW*PW]
    cplx* Linv;   // [batch][PW*PW]
    int* ipiv;    // [batch][b]
    int* idx;     // [batch][b]
    int2* moves;  // [ceil(b / PW)][batch][2 PW]  net row moves of every panel (zinv_rows.cu)
};
InvWs carve(void* ws, int b, int batch) {
    InvWs o;
    unsigned char* p = (unsigned char*)ws;
    o.Rout = (cplx*)p; p += align_up((size_t)batch * OUTER_NB_MAX * b * sizeof(cplx), 256);
    o.R = (cplx*)p;    p += align_up((size_t)batch * PW * b * sizeof(cplx), 256);
    o.Pbuf = (cplx*)p; p += align_up((size_t)batch * PW * b * sizeof(cplx), 256);
    o.Dinv = (cplx*)p; p += align_up((size_t)batch * PW * PW * sizeof(cplx), 256);
    o.Linv = (cplx*)p; p += align_up((size_t)batch * PW * PW * sizeof(cplx), 256);
    o.ipiv = (int*)p;  p += align_up((size_t)batch * b * sizeof(int), 256);
    o.idx = (int*)p;   p += align_up((size_t)batch * b * sizeof(int), 256);
    o.moves = (int2*)p;
    return o;
}

}  // namespace

size_t zinv_workspace_bytes(int b, int batch) {
    if (b <= SMALL_MAX) return 256;
    return align_up((size_t)batch * OUTER_NB_MAX * b * sizeof(cplx), 256) +
           2 * align_up((size_t)batch * PW * b * sizeof(cplx), 256) +
           2 * align_up((size_t)batch * PW * PW * sizeof(cplx), 256) +
           2 * align_up((size_t)batch * b * sizeof(int), 256) +
           align_up((size_t)((b + PW - 1) / PW) * batch * 2 * PW * sizeof(int2), 256);
}

// ---- scratch of the no-allocation entry point (negf_zinverse_batched_static, end of this file) ----------------
// One file-scope device array per GPU that loads the library, held until the process exits.  In HOST code the name
// `zinv_static_scratch` is only a stand-in for the symbol, not a device address: the address the kernels get is the
// one cudaGetSymbolAddress returns, taken once per device at set-up (negf_create, with that device current).
static __device__ __align__(256) unsigned char zinv_static_scratch[NEGF_STATIC_SCRATCH_BYTES];
constexpr int ZINV_STATIC_MAX_DEVICES = 64;
static void* zinv_static_ptr[ZINV_STATIC_MAX_DEVICES];      // [device] -> device address of that GPU's copy

static int zinv_static_setup(negf_ctx* ctx) {
    if (ctx->device < 0 || ctx->device >= ZINV_STATIC_MAX_DEVICES) return NEGF_OK;    // the entry point reports it
    void* ptr = nullptr;
    NEGF_CUDA_CHECK(ctx, cudaGetSymbolAddress(&ptr, zinv_static_scratch));
    zinv_static_ptr[ctx->device] = ptr;      // same value from every context of the device
    return NEGF_OK;
}

// shared-memory opt-ins of the blocked path, once per context (= per device) at negf_create
int zinv_prepare(negf_ctx* ctx) {
    NEGF_CUDA_CHECK(ctx, cudaFuncSetAttribute(gj_panel_cluster_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                              (int)(PANEL_SMEM_ROWS_BYTES + PANEL_SMEM_FIXED)));
    NEGF_CUDA_CHECK(ctx, cudaFuncSetAttribute(gj_dmma_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)gjd_smem_bytes<1>()));
    NEGF_CUDA_CHECK(ctx, cudaFuncSetAttribute(gj_dmma_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)gjd_smem_bytes<2>()));
    NEGF_CUDA_CHECK(ctx, cudaFuncSetAttribute(gj_colperm_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
    NEGF_CUDA_CHECK(ctx, cudaFuncSetAttribute(gj_panel_reg_kernel<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)reg_panel_smem_bytes(8)));
    NEGF_CUDA_CHECK(ctx, cudaFuncSetAttribute(gj_panel_reg_kernel<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)reg_panel_smem_bytes(16)));
    NEGF_TRY(zinv_static_setup(ctx));
    return NEGF_OK;
}

int zinv_launch(negf_ctx* ctx, int b, cplx* A, long long sA, int batch, void* ws, int* info,
                int info_code, const int* skip, const int* code_dev) {
    ProfScope _ps(ctx, NEGF_PROF_INVERSE);
    if (b <= 0 || batch <= 0) return NEGF_OK;
    if (b > 16 && b <= 64 && ctx->inv_tensor) {     // at b <= 16 the two kernels are level (15 us); the register one stays
        if (b <= 32) NEGF_CUDA_CHECK(ctx, launch_chain(ctx, gj_dmma_kernel<1>, dim3(batch), dim3(GJD_NT), gjd_smem_bytes<1>(), A, sA, b, info, info_code, skip, code_dev));
        else         NEGF_CUDA_CHECK(ctx, launch_chain(ctx, gj_dmma_kernel<2>, dim3(batch), dim3(GJD_NT), gjd_smem_bytes<2>(), A, sA, b, info, info_code, skip, code_dev));
        NEGF_LAUNCH_CHECK(ctx);
        return NEGF_OK;
    }
    if (b <= SMALL_MAX) {
        // 16 warps per matrix: half the instructions per warp and column of an 8-warp layout (the
        // kernel is bound by the per-warp dependent instruction chain, not by issue slots or FP64)
        if (b <= 16)      gj_reg_kernel<1, 1, 16><<<batch, 512, 0, ctx->stream>>>(A, sA, b, info, info_code, skip, code_dev);
        else if (b <= 32) gj_reg_kernel<1, 2, 16><<<batch, 512, 0, ctx->stream>>>(A, sA, b, info, info_code, skip, code_dev);
        else if (b <= 48) gj_reg_kernel<2, 3, 16><<<batch, 512, 0, ctx->stream>>>(A, sA, b, info, info_code, skip, code_dev);
        else if (b <= 64) gj_reg_kernel<2, 4, 16><<<batch, 512, 0, ctx->stream>>>(A, sA, b, info, info_code, skip, code_dev);
        else if (b <= 80) gj_reg_kernel<3, 5, 16><<<batch, 512, 0, ctx->stream>>>(A, sA, b, info, info_code, skip, code_dev);
        else              gj_reg_kernel<3, 6, 16><<<batch, 512, 0, ctx->stream>>>(A, sA, b, info, info_code, skip, code_dev);
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
    const size_t fixed = PANEL_SMEM_FIXED;
    const cplx one = cmake(1.0, 0.0), mone = cmake(-1.0, 0.0), zero = cmake(0.0, 0.0);
    // Two-level blocking.  Inside an outer block K = [K0, K0 + nbk) the width-w panels are
    // eliminated with their row swaps and rank-w updates restricted to the columns of K, so that
    // those columns end up holding Q = E[:, K] of the accumulated transform E (identity outside the
    // columns K); every other column then gets all nbk swaps at once and ONE rank-nbk update
    // M[:, ~K] = (M with rows K zeroed)[:, ~K] + Q R, R = the pivot rows: a GEMM with k = 128.
    // look-ahead over the outer blocks (side stream): only where the inverse runs on the caller's own stream (b above
    // the two-sided regime), outside profiling (intervals must not overlap) and with at least three outer blocks
    const int OUTER_NB = outer_nb(ctx, b, batch);
    cudaStream_t main_stream = ctx->stream;
    const bool lookahead = gj_panel_rows_supported(b) && ctx->inv_panel && ctx->inv_lookahead && !ctx->prof_on &&
                           b > 2 * OUTER_NB && ctx->inv_side != nullptr;
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
        if (gj_panel_rows_supported(b) && ctx->inv_panel) {
            // Gauss-Jordan of the panel on ALL rows, one row per thread (zinv_rows.cu): leaves the complete transform
            // columns [-T D^-1 ; D^-1 ; -B D^-1] in place and LAPACK-style pivots in ipiv
            const long long mstride = (long long)batch * 2 * PW;
            int2* mv = W.moves + (size_t)(k0 / PW) * mstride;
            RowsArgs ra{A, sA, b, k0, wk, W.ipiv, info, info_code, skip, code_dev, mv};
            NEGF_TRY(gj_panel_rows_launch(ctx, ra, batch));
            if (nbk > wk)      // the panel's exchanges on the other columns of K; pivot rows -> R, zeroed
                NEGF_TRY(gj_moves_extract_launch(ctx, A, sA, b, batch, mv, mstride, 1, k0, wk, K0, K1, k0, k0 + wk, W.R, skip));
            // M[:, other columns of K] += P' R, P' read from the panel's own columns
            // (the columns before and after the panel: ONE launch, two members of different widths)
            g.alpha = one; g.beta = one; g.m = b; g.k = wk; g.A = A + k0; g.lda = b; g.sA = sA;
            g.ldb = b; g.sB = (long long)wk * b; g.ldc = b; g.sC = sA; g.sD = sA;
            GemmGroup upd; upd.ng = 0; upd.ragged_n = 1;
            if (k0 > K0) {
                g.n = k0 - K0; g.B = W.R + K0; g.C = A + K0; g.D = A + K0;
                upd.g[upd.ng++] = g;
            }
            if (k0 + wk < K1) {
                g.n = K1 - k0 - wk; g.B = W.R + k0 + wk; g.C = A + k0 + wk; g.D = A + k0 + wk;
                upd.g[upd.ng++] = g;
            }
            if (upd.ng) NEGF_TRY(zgemm_launch_group(ctx, upd));
            continue;
        }
        if (reg_panel) {
            // one row per thread in registers; finishes P' (diagonal block and below) in place
            // rows per warp (16 warps per CTA): up to 256 rows stay in ONE CTA (no cluster barrier)
            const int R = (rows <= 128 || (rows > 256 && rows <= 1024)) ? 8 : 16;
            const int C = (rows + PNL_WARPS * R - 1) / (PNL_WARPS * R);
            PanelArgs pa{A, sA, b, k0, wk, 0, W.ipiv, W.Dinv, W.Linv, info, info_code, skip};
            cfg.gridDim = dim3(C, batch); cfg.blockDim = dim3(PNL_WARPS * 32);
            cfg.dynamicSmemBytes = reg_panel_smem_bytes(R);
            at[0].val.clusterDim.x = C;
            if (R == 8) NEGF_CUDA_CHECK(ctx, cudaLaunchKernelEx(&cfg, gj_panel_reg_kernel<8>, pa));
            else        NEGF_CUDA_CHECK(ctx, cudaLaunchKernelEx(&cfg, gj_panel_reg_kernel<16>, pa));
            NEGF_COUNT_LAUNCH(ctx);
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
                g.c_aliases_a = 1;         // tile with BN >= wk: one CTA owns all wk columns of its rows
                NEGF_TRY(zgemm_launch(ctx, g));
                g.c_aliases_a = 0;
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
        NEGF_COUNT_LAUNCH(ctx);
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
      if (lookahead) {
          // Look-ahead: the columns of the NEXT outer block get this block's swaps and rank-128 update first, on the
          // caller's stream; all other columns follow on a side stream while the caller's stream already eliminates
          // the panels of the next block (latency-bound, few CTAs) - the two touch disjoint columns.
          const long long mstride = (long long)batch * 2 * PW;
          const int2* mv0 = W.moves + (size_t)(K0 / PW) * mstride;
          const int nph = (nbk + PW - 1) / PW, K1n = min(K1 + OUTER_NB, b);
          GemmArgs g;
          g.opA = 0; g.opB = 0; g.alpha = one; g.beta = one; g.batch = batch; g.skip = skip;
          g.batch2 = 1; g.sA2 = g.sB2 = g.sD2 = g.sC2 = 0; g.alpha_vec = nullptr;
          g.m = b; g.k = nbk; g.A = A + K0; g.lda = b; g.sA = sA;
          g.ldb = b; g.sB = (long long)nbk * b; g.ldc = b; g.sC = sA; g.sD = sA;
          if (K0 > 0) NEGF_CUDA_CHECK(ctx, cudaStreamWaitEvent(main_stream, ctx->ev_inv_side, 0));   // the rest of block J-1
          if (K1 < b) {
              NEGF_TRY(gj_moves_extract_launch(ctx, A, sA, b, batch, mv0, mstride, nph, K0, nbk, K1, K1n, 0, 0, W.Rout, skip));
              g.n = K1n - K1; g.B = W.Rout + K1; g.C = A + K1; g.D = A + K1;
              NEGF_TRY(zgemm_launch(ctx, g));
          }
          NEGF_CUDA_CHECK(ctx, cudaEventRecord(ctx->ev_inv_main, main_stream));
          NEGF_CUDA_CHECK(ctx, cudaStreamWaitEvent(ctx->inv_side, ctx->ev_inv_main, 0));
          ctx->stream = ctx->inv_side;
          int rc = gj_moves_extract_launch(ctx, A, sA, b, batch, mv0, mstride, nph, K0, nbk, 0, b, K0, K1n, W.Rout, skip);
          if (rc == NEGF_OK && K0 > 0) { g.n = K0; g.B = W.Rout; g.C = A; g.D = A; rc = zgemm_launch(ctx, g); }
          if (rc == NEGF_OK && K1n < b) { g.n = b - K1n; g.B = W.Rout + K1n; g.C = A + K1n; g.D = A + K1n; rc = zgemm_launch(ctx, g); }
          cudaError_t ce = cudaEventRecord(ctx->ev_inv_side, ctx->inv_side);
          ctx->stream = main_stream;
          if (rc != NEGF_OK) return rc;
          NEGF_CUDA_CHECK(ctx, ce);
          if (K1 >= b) NEGF_CUDA_CHECK(ctx, cudaStreamWaitEvent(main_stream, ctx->ev_inv_side, 0));    // join before the epilogue
          continue;
      }
      // all nbk swaps of this outer block on the columns outside K; pivot rows -> Rout, zeroed in A
      if (gj_panel_rows_supported(b) && ctx->inv_panel) {
          const long long mstride = (long long)batch * 2 * PW;
          NEGF_TRY(gj_moves_extract_launch(ctx, A, sA, b, batch, W.moves + (size_t)(K0 / PW) * mstride, mstride,
                                           (nbk + PW - 1) / PW, K0, nbk, 0, b, K0, K1, W.Rout, skip));
      } else {
          gj_swap_extract_kernel<<<dim3((b + 127) / 128, batch), 128, 0, ctx->stream>>>(
              A, sA, b, K0, nbk, 0, b, K0, K1, W.ipiv, W.Rout, skip);
          NEGF_LAUNCH_CHECK(ctx);
      }
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
    if (b > SMALL_MAX) ctx->sweep_valid = false;     // the scratch below overlays the retained sweep state
    return zinv_launch(ctx, b, (cplx*)A, stride, batch, ctx->ws, info, 0, nullptr);
}

// No-allocation variant (include/negf.h): same kernels and launch sequence as negf_zinverse_batched, with the K1
// scratch (pivot rows, row-move tables, pivot indices) in this file's static device array instead of the context
// workspace.  Nothing in the scratch has to start at zero: every region is written by the call before it is read.
extern "C" int negf_zinverse_batched_static(negf_ctx* ctx, int b, negf_c128* A, long long stride, int batch, int* info) {
    if (!ctx || !A || b < 1 || batch < 0) return NEGF_EINVAL;
    if (ctx->prof_on) return NEGF_EUNSUPPORTED;          // the per-class profiler creates CUDA events
    if (ctx->device < 0 || ctx->device >= ZINV_STATIC_MAX_DEVICES || !zinv_static_ptr[ctx->device]) return NEGF_EUNSUPPORTED;
    if (b > SMALL_MAX && (batch > 65535 || zinv_workspace_bytes(b, batch) > (size_t)NEGF_STATIC_SCRATCH_BYTES))
        return NEGF_ESTATICLIMIT;
    if (info) NEGF_CUDA_CHECK(ctx, cudaMemsetAsync(info, 0, sizeof(int) * batch, ctx->stream));
    return zinv_launch(ctx, b, (cplx*)A, stride, batch, zinv_static_ptr[ctx->device], info, 0, nullptr);
}
