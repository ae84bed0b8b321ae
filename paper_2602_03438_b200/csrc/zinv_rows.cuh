// Row-per-thread Gauss-Jordan panel kernel of the blocked inverse (zinv_rows.cu), called from zinv.cu.
#pragma once
#include "common.cuh"

struct RowsArgs {
    cplx* A; long long sA;     // [batch] matrices b x b, row-major, stride sA
    int b, k0, w;              // panel = columns [k0, k0 + w), w <= 32
    int* ipiv;                 // [batch][b]: ipiv[k] = row exchanged with row k at step k (LAPACK style)
    int* info; int code;       // info[e] = code (or column + 1 when code <= 0) on a zero pivot, first failure wins
    const int* skip;           // optional [batch]: entry skipped when != 0
    const int* code_dev;       // optional device int added to code (iteration counter of the decimation WHILE graph)
    // net effect of the panel's row exchanges as independent moves: moves[e][2 j] = (k0 + j, source row),
    // moves[e][2 j + 1] = (partner position of step j, source row): "position dst now holds what row src held
    // before the panel" (duplicates agree).  [batch][2 * 32] int2; lets the other columns be permuted in parallel
    int2* moves;
};
// Applies the exchanges of `nphase` consecutive panels (moves lists of 2 * 32 entries, `moves_stride` int2 apart;
// np pivots in all, 32 per panel but the last) to
// the columns [clo, chi) except [xlo, xhi) of every matrix, then moves rows p0 .. p0 + np - 1 to R [batch][np][b]
// and zeroes them in A - all loads of a phase before its stores, no dependent chain of swaps.
int gj_moves_extract_launch(negf_ctx* ctx, cplx* A, long long sA, int b, int batch, const int2* moves,
                            long long moves_stride, int nphase, int p0, int np, int clo, int chi,
                            int xlo, int xhi, cplx* R, const int* skip);
bool gj_panel_rows_supported(int b);
// enqueues the panel kernel on ctx->stream (thread-block cluster of ceil(b / 256) CTAs per matrix)
int gj_panel_rows_launch(negf_ctx* ctx, const RowsArgs& a, int batch);
