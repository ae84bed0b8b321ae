// Carve-up of the caller-owned workspace (negf_set_workspace), shared by all calls.
#pragma once
#include "common.cuh"

constexpr int NEGF_NSCRATCH = 13;   // decimation needs 13 blocks per energy, the sweeps 9
constexpr int NEGF_PAIR_MAX_B = 128; // up to this block size both leads are decimated in ONE batch of 2*NE entries
inline int negf_tmul(int b) { return b <= NEGF_PAIR_MAX_B ? 2 : 1; }

struct Workspace {
    cplx* g;        // [NE][n][b][b]    left-connected g_i        (retained sweep state)
    cplx* X;        // [NE][n-1][b][b]  X_i = g_i A_{i,i+1}       (retained)
    cplx* Y;        // [NE][n-1][b][b]  Y_i = A_{i+1,i} g_i       (retained)
    cplx* gx;       // [NE][n][b][b]    left-connected g^x_i (one of </> at a time)
    cplx* Z;        // [NE][n-1][b][b]  Z_i = g_i A_{i,i-1} (S5), then T2_i (S6)
    cplx* Q;        // [NE][n][b][b]    S5 temporaries, then Q_i when G^x_upper is not requested
    cplx* Aup;      // [NE][n-1][b][b]  A_{i,i+1}, only when S != I or Sigma^R_S is BT   (retained)
    cplx* Alow;     // [NE][n-1][b][b]  A_{i+1,i}, likewise                              (retained)
    cplx* T[NEGF_NSCRATCH];   // [NE][b][b] each
    void* inv;      // zinv workspace (batch NE * tmul)
    void* inv2;     // second zinv workspace (batch NE) for the chain that runs on a side stream
    void* inv_side(bool side) const { return side ? inv2 : inv; }
    double* ref;    // [NE]
    int* done;      // [NE]
    int* sing;      // [NE]
    int* tmpinfo;   // [NE]
    int* its;       // [2 NE] doublings done
    double* acc;    // [2 NE][128][2] partial sums of squares of the fused Sancho-Rubio step
    unsigned* ticket;  // [2 NE]
    size_t bytes;
};

// Aup / Alow sit at the END so that every other offset is independent of `assembled`.
inline Workspace carve_workspace(void* base, int n, int b, int ne, bool assembled = false) {
    Workspace w;
    unsigned char* p = (unsigned char*)base;
    const size_t blk = (size_t)b * b * sizeof(cplx);
    auto take = [&](size_t nbytes) { unsigned char* r = p; p += align_up(nbytes, 256); return r; };
    w.g = (cplx*)take(blk * n * ne);
    w.X = (cplx*)take(blk * (n > 1 ? n - 1 : 0) * ne);
    w.Y = (cplx*)take(blk * (n > 1 ? n - 1 : 0) * ne);
    w.gx = (cplx*)take(blk * n * ne);
    w.Z = (cplx*)take(blk * (n > 1 ? n - 1 : 0) * ne);
    w.Q = (cplx*)take(blk * n * ne);
    const int tm = negf_tmul(b);
    for (int t = 0; t < NEGF_NSCRATCH; t++) w.T[t] = (cplx*)take(blk * ne * tm);
    w.inv = take(zinv_workspace_bytes(b, ne * tm));
    w.inv2 = tm == 2 ? take(zinv_workspace_bytes(b, ne)) : w.inv;
    w.ref = (double*)take(sizeof(double) * ne * 2);
    w.done = (int*)take(sizeof(int) * ne * 2);
    w.sing = (int*)take(sizeof(int) * ne * 2);
    w.tmpinfo = (int*)take(sizeof(int) * ne * 2);
    w.its = (int*)take(sizeof(int) * ne * 2);
    w.acc = (double*)take(sizeof(double) * ne * 2 * 2 * 128);      // [2 NE][SR_SPLIT_MAX][2] (elementwise.cu)
    w.ticket = (unsigned*)take(sizeof(unsigned) * ne * 2);
    w.Aup = w.Alow = nullptr;
    if (assembled) {
        w.Aup = (cplx*)take(blk * (n > 1 ? n - 1 : 0) * ne);
        w.Alow = (cplx*)take(blk * (n > 1 ? n - 1 : 0) * ne);
    }
    w.bytes = (size_t)(p - (unsigned char*)base);
    return w;
}
