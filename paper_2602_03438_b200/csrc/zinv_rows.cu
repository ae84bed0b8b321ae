// K1, blocked path (b > 96), step 1: Gauss-Jordan of one width-32 panel on ALL rows of the matrix, one matrix
// ROW PER THREAD (every g_i of the RGF forward sweep, and every g = a_b^-1 of the
// Sancho-Rubio doubling at b > 96 spends its sequential time here).
//
// The first panel kernel of this path (zinv.cu: lane = panel column, R rows per warp in registers) needs ~830
// warp instructions per warp and column: every warp scans / selects / exchanges over its rows with half of the
// lanes idle, 4-5 us per column, 150 us per panel.  Here a thread owns one row of the panel, its 32 columns in
// registers; the column being eliminated always sits in register 0 and the row is rotated by one register per
// step (rows_step), so every register index is a constant although the column loop is a real loop:
//   * pivot of column J: partial pivoting on the leading 32 bits of |re|+|im| (sign, exponent, 20 mantissa bits)
//     among the rows at or below the panel that were not pivots yet, lowest row first among equals: one
//     redux.sync + one ballot per warp, one block barrier for the CTA's candidate, whose row is pushed to every
//     CTA of the cluster (DSMEM) together with its key, ONE cluster barrier, and everybody knows the pivot row;
//   * pivoting inside the panel is IMPLICIT (rows never leave their thread); the row exchanges LAPACK would do
//     (ipiv[k] = position of the pivot row at step k) are replayed on an index table by one thread per CTA and
//     applied when the rows are written back, so the other kernels of the blocked inverse (row swaps on the other
//     columns, final column permutation) see the usual sequential-swap pivots;
//   * elimination: row_i -= (x_i[J] / pivot) * pivot row on all 31 other columns: 124 DFMA per thread and column
//     from registers and broadcast shared-memory reads - every lane busy.
// The rows ABOVE the panel take part too (they are only excluded from the pivot search), so the kernel leaves
// the complete transform columns E[:, K] = [-T D^-1 ; D^-1 ; -B D^-1] in place and the separate product
// P' = -T Dinv of the first version is gone.  Up to 8 x 256 = 2048 rows per matrix (cluster of up to 8 CTAs).
#include <cooperative_groups.h>

#include "common.cuh"
#include "zinv_rows.cuh"

namespace cg = cooperative_groups;

namespace {

constexpr int RW = 32;            // panel width
constexpr int RNT = 256;          // rows = threads per CTA
constexpr int RCMAX = 8;          // portable cluster size
constexpr int RNONE = 0x7fffffff;
constexpr unsigned FULL = 0xffffffffu;

struct RowsSmem {
    cplx candrow[2][RCMAX][RW];                 // [parity][rank]: the candidate row of every CTA of the cluster
    cplx rowbuf[RNT / 32][RW];                  // staging of a warp's candidate row
    unsigned cand_key[2][RCMAX]; int cand_row[2][RCMAX];
    unsigned wkey[2][RNT / 32]; int wrow[2][RNT / 32];
    int at[RCMAX * RNT];                        // at[position] = original row now there (replayed exchanges)
    int where[RCMAX * RNT];                     // where[original row] = its position
    int partner[RW];                            // position exchanged with k0 + J at step J
};

// 1 / a for a pivot: hardware reciprocal estimate + two Newton steps (as in zinv.cu)
__device__ __forceinline__ cplx rows_recip(cplx a) {
    const double x = fma(a.x, a.x, a.y * a.y);
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    double e = fma(-x, r, 1.0);
    r = fma(r, e, r);
    e = fma(-x, r, 1.0);
    r = fma(r, e, r);
    return cmake(a.x * r, -a.y * r);
}

// One Gauss-Jordan step on panel column J (a RUNTIME index): the column to eliminate is ALWAYS register 0 of `x`;
// the updated row leaves in `y` rotated left by one (y[c-1] = new x[c], y[31] = the transform column), so the
// next step finds its column in register 0 again.  The rotation costs nothing (it is the destination register of
// the DFMAs) and makes the body of the column loop the same code for every column: two steps (x -> y, y -> x) are
// the whole loop body, ~13 KB of SASS that stays in the instruction cache.  (Unrolling all 32 columns with
// constant register indices gave 24 000 instructions of straight-line code, each executed once per warp and
// panel: instruction-fetch bound, 3-4 us per column.)  Every thread rotates alike, so the candidate rows pushed
// through shared memory are in the same rotated order.
template <int PAR>
__device__ __forceinline__ void rows_step(const cplx (&x)[RW], cplx (&y)[RW], bool& used, RowsSmem& S, const RowsArgs& a,
                                          const int J, const int e, const int i, const int rank, const int C,
                                          cg::cluster_group& cluster, const int warp, const int lane) {
    // ---- candidate of this warp, of this CTA
    const bool elig = !used && i >= a.k0 && i < a.b;
    unsigned key = 0u;
    if (elig) key = (unsigned)((unsigned long long)__double_as_longlong(cabs1(x[0])) >> 32) + 1u;
    const unsigned wmax = __reduce_max_sync(FULL, key);
    const unsigned bal = __ballot_sync(FULL, elig && key == wmax);
    if (lane == 0) {
        S.wkey[PAR][warp] = wmax;
        S.wrow[PAR][warp] = bal ? i + (__ffs(bal) - 1) : RNONE;       // lane 0 holds row i, lane l row i + l
    }
    __syncthreads();
    unsigned ck = 0u; int cw = 0;
#pragma unroll
    for (int q = 0; q < RNT / 32; q++) {
        const unsigned k2 = S.wkey[PAR][q];
        if (k2 > ck) { ck = k2; cw = q; }                              // rows ascend with the warp: lowest row wins ties
    }
    const int crow = ck ? S.wrow[PAR][cw] : RNONE;
    if (warp == cw) {                           // (no candidate at all: warp 0 pushes the empty key)
        if (i == crow) {
#pragma unroll
            for (int c = 0; c < RW; c++) S.rowbuf[warp][c] = x[c];
        }
        __syncwarp();
        const cplx v = S.rowbuf[warp][lane];
        if (C == 1) {
            S.candrow[PAR][0][lane] = v;
            if (lane == 0) { S.cand_key[PAR][0] = ck; S.cand_row[PAR][0] = crow; }
        } else {
            for (int q = 0; q < C; q++) {
                RowsSmem* R = cluster.map_shared_rank(&S, q);
                R->candrow[PAR][rank][lane] = v;
                if (lane == 0) { R->cand_key[PAR][rank] = ck; R->cand_row[PAR][rank] = crow; }
            }
        }
    }
    if (C == 1) __syncthreads(); else cluster.sync();
    // ---- the pivot row: largest key, lowest row among equals (rows ascend with the rank)
    unsigned wk = 0u; int prow = RNONE, wq = 0;
    for (int q = 0; q < C; q++) {
        const unsigned k2 = S.cand_key[PAR][q];
        if (k2 > wk) { wk = k2; prow = S.cand_row[PAR][q]; wq = q; }
    }
    const bool sing = wk <= 1u;                 // every candidate is zero in its leading 32 bits (or none left)
    const cplx* pr = S.candrow[PAR][wq];
    const cplx d = sing ? cmake(1.0, 0.0) : rows_recip(pr[0]);
    if (threadIdx.x == 0 && prow != RNONE) {    // replay LAPACK's exchange of positions k0 + J and where[prow]
        const int pj = a.k0 + J;
        const int q = S.where[prow], o = S.at[pj];
        S.at[pj] = prow; S.where[prow] = pj; S.at[q] = o; S.where[o] = q;
        S.partner[J] = q;
        if (rank == 0) {
            a.ipiv[(size_t)e * a.b + pj] = q;
            if (sing && a.info && a.info[e] == 0) a.info[e] = a.code > 0 ? a.code + (a.code_dev ? *a.code_dev : 0) : pj + 1;
        }
    }
    // ---- elimination on all other columns of the panel; the eliminated column becomes the transform column
    if (i == prow) {
        used = true;
#pragma unroll
        for (int c = 1; c < RW; c++) y[c - 1] = cmul(x[c], d);
        y[RW - 1] = d;
    } else {
        const cplx m = cmul(x[0], d);
#pragma unroll
        for (int c = 1; c < RW; c++) { cplx t = x[c]; cfms(t, m, pr[c]); y[c - 1] = t; }
        y[RW - 1] = cneg(m);
    }
}

__global__ void __launch_bounds__(RNT, 1) gj_panel_rows_kernel(const RowsArgs a) {
    cg::cluster_group cluster = cg::this_cluster();
    const int rank = (int)cluster.block_rank();
    const int C = (int)cluster.num_blocks();
    const int e = blockIdx.y;
    if (a.skip && a.skip[e]) return;                    // uniform over the cluster
    __shared__ RowsSmem S;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int i = rank * RNT + tid;                     // my row of the matrix
    cplx* g = a.A + (size_t)e * a.sA + a.k0;            // panel origin (row 0)
    cplx x[RW], y[RW];
#pragma unroll
    for (int c = 0; c < RW; c++)
        x[c] = (i < a.b && c < a.w) ? g[(size_t)i * a.b + c] : cmake(0.0, 0.0);
    for (int p = tid; p < C * RNT; p += RNT) { S.at[p] = p; S.where[p] = p; }
    bool used = false;
    __syncthreads();
    int J = 0;
#pragma unroll 1
    for (; J + 1 < a.w; J += 2) {
        rows_step<0>(x, y, used, S, a, J, e, i, rank, C, cluster, warp, lane);
        rows_step<1>(y, x, used, S, a, J + 1, e, i, rank, C, cluster, warp, lane);
    }
    if (J < a.w) {                                      // odd width (ragged last panel)
        rows_step<0>(x, y, used, S, a, J, e, i, rank, C, cluster, warp, lane);
#pragma unroll
        for (int c = 0; c < RW; c++) x[c] = y[c];
    }
    __syncthreads();
    // after w steps panel column c sits in register 32 - w + c; the row goes to position where[i] (replayed exchanges)
    if (rank == 0 && a.moves && tid < a.w) {           // the exchanges as independent moves, for the other columns
        int2* mv = a.moves + (size_t)e * 2 * RW;
        const int q = S.partner[tid];
        mv[2 * tid] = make_int2(a.k0 + tid, S.at[a.k0 + tid]);
        mv[2 * tid + 1] = make_int2(q, S.at[q]);
    }
    if (i < a.b) {
        cplx* orow = g + (size_t)S.where[i] * a.b;
        const int shift = RW - a.w;
#pragma unroll
        for (int r = 0; r < RW; r++)
            if (r >= shift) orow[r - shift] = x[r];
    }
    if (C > 1) cluster.sync();                          // nobody exits while remote shared memory may still be targeted
}

// permutes the other columns by the panels' move lists (see zinv_rows.cuh); block = 32 columns x 8 move lanes
constexpr int MV_COLS = 32, MV_LANES = 8;
__global__ void __launch_bounds__(MV_COLS * MV_LANES) gj_moves_extract_kernel(
    cplx* A, long long sA, int b, const int2* moves, long long moves_stride, int nphase, int p0, int np,
    int clo, int chi, int xlo, int xhi, cplx* R, const int* skip) {
    const int e = blockIdx.y;
    if (skip && skip[e]) return;
    __shared__ cplx sm[2 * RW][MV_COLS];
    __shared__ int2 smv[2 * RW];
    const int tx = threadIdx.x, ty = threadIdx.y;
    // column of this thread, the excluded range [xlo, xhi) skipped
    int c = clo + blockIdx.x * MV_COLS + tx;
    if (c >= xlo) c += xhi - xlo;
    const bool live = c < chi;
    cplx* g = A + (size_t)e * sA;
    int left = np;
    for (int ph = 0; ph < nphase; ph++) {
        const int w = min(RW, left);
        left -= w;
        const int2* mv = moves + (size_t)e * 2 * RW + (size_t)ph * moves_stride;
        const int t = ty * MV_COLS + tx;
        if (t < 2 * w) smv[t] = mv[t];
        __syncthreads();
        for (int m = ty; m < 2 * w; m += MV_LANES) if (live) sm[m][tx] = g[(size_t)smv[m].y * b + c];
        __syncthreads();
        for (int m = ty; m < 2 * w; m += MV_LANES) if (live) g[(size_t)smv[m].x * b + c] = sm[m][tx];
        __syncthreads();
    }
    if (!live) return;
    cplx* r = R + (size_t)e * np * b;
    for (int j = ty; j < np; j += MV_LANES) {
        r[(size_t)j * b + c] = g[(size_t)(p0 + j) * b + c];
        g[(size_t)(p0 + j) * b + c] = cmake(0.0, 0.0);
    }
}

}  // namespace

int gj_moves_extract_launch(negf_ctx* ctx, cplx* A, long long sA, int b, int batch, const int2* moves,
                            long long moves_stride, int nphase, int p0, int np, int clo, int chi,
                            int xlo, int xhi, cplx* R, const int* skip) {
    const int ncols = (chi - clo) - (xhi - xlo);
    if (ncols <= 0 || batch <= 0) return NEGF_OK;
    gj_moves_extract_kernel<<<dim3((ncols + MV_COLS - 1) / MV_COLS, batch), dim3(MV_COLS, MV_LANES), 0, ctx->stream>>>(
        A, sA, b, moves, moves_stride, nphase, p0, np, clo, chi, xlo, xhi, R, skip);
    NEGF_LAUNCH_CHECK(ctx);
    return NEGF_OK;
}

bool gj_panel_rows_supported(int b) { return b <= RCMAX * RNT; }

int gj_panel_rows_launch(negf_ctx* ctx, const RowsArgs& a, int batch) {
    if (a.w < 1 || a.w > RW || !gj_panel_rows_supported(a.b)) return NEGF_EINVAL;
    const int C = (a.b + RNT - 1) / RNT;
    cudaLaunchConfig_t cfg = {};
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = C; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1; cfg.stream = ctx->stream;
    cfg.gridDim = dim3(C, batch); cfg.blockDim = dim3(RNT); cfg.dynamicSmemBytes = 0;
    NEGF_CUDA_CHECK(ctx, cudaLaunchKernelEx(&cfg, gj_panel_rows_kernel, a));
    NEGF_COUNT_LAUNCH(ctx);
    return NEGF_OK;
}
