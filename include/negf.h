/*
 * negf.h - C ABI of the B200-native LSE+OBC hot path of arxiv/paper_2602_03438.
 *
 * Path (Fig. 1 red blocks "LSE+OBC"; Eqs. 1-2):
 * for many independent energies E, with z = E + i*eta and the block-tridiagonal (BT)
 *     A(E) = z S - H - Sigma^R_B - Sigma^R_S,
 * compute the selected blocks (i,i), (i,i+1), (i+1,i) of
 *     G^R  = A^-1                                   (Eq. 1)
 *     G^<> = G^R (Sigma^<>_B + Sigma^<>_S) (G^R)^H  (Eq. 2)
 * by the recursive Green's function (RGF) sweeps, with the open-boundary
 * self-energies Sigma_B ("open boundary condition term") obtained by
 * Sancho-Rubio decimation of the lead blocks (BASELINE.json:north_star),
 * and reduce them to density, LDOS, transmission and currents.
 *
 * Conventions
 *  - negf_c128 = interleaved (re, im) doubles.  Every block is dense b x b ROW-MAJOR with
 *    leading dimension b; blocks of a family are contiguous; batched arrays are
 *    [N_E][n or n-1][b][b] (energy slowest).  No padding.
 *  - Unless a parameter says HOST, every array pointer is a DEVICE pointer owned by the
 *    caller.  The library never allocates or frees caller arrays; its only own allocation
 *    is the small context object.  Scratch memory is the caller-provided workspace.
 *  - All calls enqueue work on the context's stream and return without synchronising
 *    (exception: negf_pipeline_host and negf_fp64_peak, which say so).
 *  - Return value: 0 = enqueued; negative = argument / runtime error (see negf_strerror).
 *    Numerical failures are reported PER ENERGY in the device int arrays info/status:
 *    0 ok; k > 0 = zero pivot while inverting block k-1 (for the decimation: iteration k);
 *    -1 = decimation hit max_iter without meeting tol (result still written).
 *  - There is no CPU fallback: every call needs a CUDA device of compute capability 10.0.
 *  - Thread safety: one context per host thread / stream.
 */
#ifndef NEGF_H
#define NEGF_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct { double re, im; } negf_c128;
typedef struct negf_ctx negf_ctx;

/* error codes */
#define NEGF_OK            0
#define NEGF_EINVAL       -1   /* bad argument (NULL where required, n < 1, side not 0/1, ...) */
#define NEGF_ENOWORKSPACE -2   /* workspace missing or smaller than negf_workspace_bytes()     */
#define NEGF_EUNSUPPORTED -3   /* combination not implemented (documented at the call)         */
#define NEGF_ECUDA        -4   /* CUDA runtime error; see negf_last_cuda_error()               */
#define NEGF_ENOSTATE     -5   /* call needs the retained sweep state of negf_rgf_retarded     */
#define NEGF_ESTATICLIMIT  -6   /* problem needs more than NEGF_STATIC_SCRATCH_BYTES (negf_zinverse_batched_static) */

/* kinds of scattering self-energy Sigma_S */
#define NEGF_SIGMA_NONE   0
#define NEGF_SIGMA_SCALAR 1    /* s(E) * I on every diagonal block                            */
#define NEGF_SIGMA_BT     2    /* dense block-tridiagonal per energy                           */

/* flags of negf_rgf_retarded */
#define NEGF_KEEP_SWEEP   1    /* retain g_i, X_i, Y_i in the workspace for negf_rgf_lesser_greater */

/* Device + energy grid (A = E S - H for electrons; BT shape). */
typedef struct {
    int n_blocks;              /* n >= 1 diagonal blocks                                       */
    int block_size;            /* b >= 1                                                       */
    int n_energy;              /* N_E >= 1 energies resident in this batch                     */
    const negf_c128* H_diag;   /* [n][b][b]   Hermitian blocks, shared by all energies         */
    const negf_c128* H_upper;  /* [n-1][b][b] H_{i,i+1}; H_{i+1,i} = H_{i,i+1}^H (may be NULL if n == 1) */
    const negf_c128* S_diag;   /* [n][b][b]   or NULL: S = I (then S_upper must be NULL too)   */
    const negf_c128* S_upper;  /* [n-1][b][b] S_{i,i+1}; S_{i+1,i} = S_{i,i+1}^H               */
    const double*    energy;   /* [N_E] real energies E                                         */
    double           eta;      /* z = E + i*eta multiplies S everywhere, leads included (R1)   */
    /* Momentum (k-point) batching ("the momentum dependence is omitted for simplicity"; SURVEY.md
     * 8(f) item 2): n_k > 1 makes H_diag / H_upper / S_diag / S_upper arrays of n_k devices, [n_k][n][b][b] and
     * [n_k][n-1][b][b], and k_index [N_E] (DEVICE ints in [0, n_k)) names the device of every batch entry, so
     * the batch axis is any list of (k, E) pairs: one lock-step batch of N_E entries, e.g. N_k x N_E' in k-major
     * order with `energy` repeating the grid.  n_k <= 1 (or k_index NULL): one device, as above.  Every
     * per-energy array of the calls below is per batch entry.  Sums over k (density, T) are the caller's:
     * negf_observables folds weights[e] (= w_k w_E) into the density. */
    int              n_k;
    const int*       k_index;
} negf_problem;

/* One self-energy family: boundary blocks on the two contacts plus Sigma_S.
 * For the retarded Sigma^R all of diag/upper/lower are independent.
 * For Sigma^< and Sigma^> the full matrix is anti-Hermitian: lower = -upper^H is IMPLIED
 * and `lower` is ignored. */
typedef struct {
    int kind;                  /* NEGF_SIGMA_NONE | _SCALAR | _BT                              */
    const negf_c128* scalar;   /* [N_E]             (kind SCALAR)                              */
    const negf_c128* diag;     /* [N_E][n][b][b]    (kind BT)                                  */
    const negf_c128* upper;    /* [N_E][n-1][b][b]  (kind BT) Sigma_{i,i+1}                    */
    const negf_c128* lower;    /* [N_E][n-1][b][b]  (kind BT, retarded only) Sigma_{i+1,i}     */
    const negf_c128* left;     /* [N_E][b][b] boundary block added on block 0,   or NULL       */
    const negf_c128* right;    /* [N_E][b][b] boundary block added on block n-1, or NULL       */
} negf_sigma;

/* Optional explicit lead (overrides "periodic copies of the contact blocks", reading R2;
 * required when n_blocks == 1).  H_u/S_u couple a lead cell to its next cell on the right.
 * With k-point batching (negf_problem.n_k > 1) every member is [n_k][b][b]. */
typedef struct {
    const negf_c128* H_d;      /* [b][b] */
    const negf_c128* H_u;      /* [b][b] */
    const negf_c128* S_d;      /* [b][b] or NULL (identity) */
    const negf_c128* S_u;      /* [b][b] or NULL (zero)     */
} negf_lead;

/* ---- context ---------------------------------------------------------------------------- */
int negf_create(negf_ctx** out, int device);
int negf_destroy(negf_ctx* ctx);
/* cudaStream_t passed as void*; NULL = the legacy default stream. */
int negf_set_stream(negf_ctx* ctx, void* cuda_stream);
/* Bytes of workspace needed by ANY call on this problem shape (kind_max = the richest
 * Sigma kind that will be passed, flags as for negf_rgf_retarded). */
int negf_workspace_bytes(const negf_problem* p, int kind_max, int flags, size_t* bytes);
/* Caller-owned device scratch (e.g. a torch tensor), 256-byte aligned. Retained sweep state
 * lives here; replacing the workspace drops it. */
int negf_set_workspace(negf_ctx* ctx, void* dev_ptr, size_t bytes);
/* Options.  NEGF_OPT_GRAPH_LOOPS (default 2): the Sancho-Rubio doublings of negf_obc_decimate[_pair] run as a
 * cached device-driven WHILE graph (CUDA conditional node) that stops when every energy has converged; 1 = only
 * for block sizes up to 96 (larger blocks: the host loop); 0 = the plain host loop of max_iter masked doublings
 * everywhere (and no cached call graphs).  Above b = 96 one masked doubling is ~300 launches of kernels that exit at
 * once (the blocked inverse), and the stopping rule is met after ~22 of max_iter = 64 doublings: the graph takes
 * 27 000 of the 42 000 launches of a configs[4] step away (12.56 -> 12.47 s; configs[3] 12.78 -> 12.61 s, configs[2]
 * 1665 -> 1637 ms).  Same arithmetic and results either way (bit-identical, tested).
 * NEGF_OPT_GEMM_3M (default 0): in the compute-bound regime (blocks above 64 that fill the machine with
 * 128-row tiles) complex products use the 3M decomposition (three real DMMA products instead of four: 25 % fewer
 * tensor-pipe instructions; the imaginary part is accurate norm-wise, not component-wise).  Off by default: the
 * 4M kernel is the one the FP64 roofline fraction is quoted on.
 * NEGF_OPT_INV_TENSOR (default 1): block sizes 17..64 are inverted by the blocked Gauss-Jordan kernel whose
 * rank-4 updates run on the FP64 tensor pipe (one CTA per matrix, same partial pivoting and the same order
 * of elimination updates per element as the unblocked kernel); 0 = the register-resident unblocked
 * Gauss-Jordan kernel for every block size up to 96 (the kernel 65..96 and 1..16 always use).  Set it
 * before the first call of a shape (cached call graphs keep the kernel they were captured with).
 * NEGF_OPT_ENERGY_GROUPS (default 0 = automatic): number of concurrent energy groups (1..4) that
 * negf_pipeline_device / negf_pipeline_host split the batch into.  K3, the energy-batch scheduler: in the
 * latency-bound small-block regime every launch of the sequential chains leaves SMs idle, so the batch runs as
 * groups of energies that walk the whole path S2-S7 concurrently on streams owned by the context (one group's
 * inversions overlap another's products); same arithmetic per energy, same outputs.  Automatic = 4 groups for
 * block sizes up to 96 with at least 32 energies, else 1 (at large blocks every launch fills the GPU).
 * NEGF_OPT_INV_PANEL (default 1): panels of the blocked inverse (97 <= b <= 2048) are eliminated by the
 * row-per-thread Gauss-Jordan kernel (all rows of the matrix, partial pivoting on the leading 32 bits of
 * |re|+|im|); 0 = the first panel kernel (LU of the rows at and below the panel, lane = panel column), which
 * larger blocks always use.  Same pivoting rule up to the key width, same results up to rounding.
 * NEGF_OPT_INV_LOOKAHEAD (default 1): the blocked inverse of blocks above 256 applies the rank-128 update of an
 * outer block to the columns of the NEXT outer block first and to all other columns on a side stream of the
 * context, while the caller's stream already eliminates the next block's panels; joined before the call
 * returns.  0 = everything in order on the caller's stream.  Bit-identical results.
 * NEGF_OPT_INV_OUTER (default 0 = automatic: 128 columns up to b = 1024, 256 above): width of the outer block of
 * the blocked inverse, i.e. the k of its big trailing updates (a multiple of 32, at most 256).
 * NEGF_OPT_FUSED_SMALL (default 1 = automatic: when N_E <= number of SMs; 2 = always; 0 = never): for block sizes
 * up to 32 the whole chain of one energy runs in ONE thread block
 * with every operand in shared memory: negf_obc_decimate[_pair] is one launch (one CTA per lead and energy walks the
 * complete doubling loop), negf_rgf_retarded one launch (one CTA per energy, forward and backward sweep),
 * negf_rgf_lesser_greater one launch (one CTA per energy and < / >).  0 = the batched lock-step launches used for
 * larger blocks.  Same definitions, results equal to rounding.  Set it before negf_rgf_retarded: the retained
 * sweep state of one regime is not valid for the other.
 * NEGF_OPT_PDL (default 1; bit 0 = on, bit 1 = also inside the decimation WHILE graph): the kernels of the
 * latency-bound chains (complex GEMM with tiles up to 32 x 32, the one-CTA inverse of 16 < b <= 64, the decimation
 * step) are launched with CUDA's programmatic-stream-serialization attribute: their CTAs are placed while the previous
 * kernel of the stream drains and block in griddepcontrol.wait until it has completed, which takes the launch gap out of
 * the dependent chain (b = 64, 64 energies, one stream: negf_rgf_retarded 1.78 -> 1.71 ms, negf_rgf_lesser_greater 2.80 ->
 * 2.69 ms).  Bit-identical results.  The concurrent energy groups of negf_pipeline_device / _host always run with 0:
 * they already cover each other's gaps, and a waiting grid would only take SM slots from the other groups (measured
 * 5.79 -> 6.12 ms per configs[1] step with it).  Changing the option drops the cached call graphs.
 * The environment variable NEGF_PDL (0..3), read by negf_create, overrides the default (developer switch to run a whole
 * test suite under one setting). */
#define NEGF_OPT_GRAPH_LOOPS   1
#define NEGF_OPT_GEMM_3M       2
#define NEGF_OPT_INV_TENSOR    3
#define NEGF_OPT_ENERGY_GROUPS 4
#define NEGF_OPT_INV_PANEL     5
#define NEGF_OPT_INV_LOOKAHEAD 6
#define NEGF_OPT_INV_OUTER     7
#define NEGF_OPT_FUSED_SMALL   8
#define NEGF_OPT_PDL           9
#define NEGF_MAX_ENERGY_GROUPS 4
int negf_set_option(negf_ctx* ctx, int option, int value);
const char* negf_strerror(int code);
/* cudaError_t of the last failing runtime call on this context (0 if none). */
int negf_last_cuda_error(const negf_ctx* ctx);
/* Number of kernels this context has launched since creation (bench.py's gpu_launches). */
long long negf_launch_count(const negf_ctx* ctx);
/* Kernels in ONE execution of the body (two doublings + the loop condition) of the cached decimation WHILE graph of
 * this context, or of its first energy group when the groups hold the graphs; 0 when no such graph exists.  The
 * graph's kernels run on the device without host launches, so negf_launch_count does not see its iterations:
 * bench.py multiplies this by the executed iterations it reads from the iteration counters. */
long long negf_obc_graph_kernels(const negf_ctx* ctx);

/* Per-kernel-class device timing for bench.py's roofline: when enabled, one CUDA event is recorded on
 * the context stream whenever the kernel class of the next launch differs from the previous one, so the
 * consecutive launches of a class form one timed interval; the side streams and the call graphs are not
 * used while profiling (every kernel runs on the caller's stream, plain launches), so intervals never
 * overlap.  Never enable it inside a timed throughput run.
 * negf_profile_read SYNCHRONISES the stream, folds all finished intervals into the per-class totals and
 * returns milliseconds and number of kernel launches of `kclass` since the last reset; reset != 0 clears the
 * totals of that class afterwards.  ms / sites may be NULL. */
#define NEGF_PROF_GEMM        0   /* K2 complex GEMM (DMMA)                                        */
#define NEGF_PROF_INVERSE     1   /* K1 inverse (all its kernels, inner GEMMs included)             */
#define NEGF_PROF_ELEMENTWISE 2   /* O(b^2) assembly / combination kernels                          */
#define NEGF_PROF_OBSERVABLES 3   /* S7 reductions                                                  */
#define NEGF_PROF_FUSED       4   /* fused small-block chain kernels                                */
#define NEGF_PROF_CLASSES     5
int negf_profile_enable(negf_ctx* ctx, int on);
int negf_profile_read(negf_ctx* ctx, int kclass, double* ms, long long* sites, int reset);

/* ---- S2: open-boundary self-energies ------------
 * For each energy: a_d = z S_d - H_d, a_u = z S_u - H_u, a_l = z S_u^H - H_u^H of the lead
 * (default: contact blocks 0/0-1 for side 0, n-1/(n-2,n-1) for side 1); Sancho-Rubio doubling
 *   g = a_b^-1; a_s -= l g u (side 0) | u g l (side 1); a_b -= u g l + l g u; u = -u g u; l = -l g l
 * until ||u||_F + ||l||_F <= tol (||a_u||_F + ||a_l||_F) or max_iter (reading R3); then
 *   g_s = a_s^-1, Sigma^R = a_l g_s a_u (side 0) | a_u g_s a_l (side 1),
 *   Gamma = i (Sigma^R - Sigma^R^H), f = 1/(1+exp((E-mu)/kT)),
 *   Sigma^< = i f Gamma, Sigma^> = -i (1-f) Gamma.
 * Outputs [N_E][b][b] each; any of gamma, sigma_lesser, sigma_greater, g_surface, fermi may be
 * NULL.  iters [N_E] = doublings done; status [N_E] as described at the top. */
int negf_obc_decimate(negf_ctx* ctx, const negf_problem* p, const negf_lead* lead /* or NULL */,
                      int side, double mu, double kT, double tol, int max_iter,
                      negf_c128* sigma_r, negf_c128* gamma,
                      negf_c128* sigma_lesser, negf_c128* sigma_greater,
                      negf_c128* g_surface, double* fermi, int* iters, int* status);

/* Both leads in one call (K3, the energy-batch scheduler): for block sizes up to 128 the left and
 * right decimations of all energies run as ONE batch of 2 N_E entries, so every launch carries
 * twice the work; above that the two leads run one after the other.  Same results as two
 * negf_obc_decimate calls.  Members of negf_obc_out as the like-named arguments above
 * (sigma_r, iters, status required; the others may be NULL). */
typedef struct {
    negf_c128 *sigma_r, *gamma, *sigma_lesser, *sigma_greater, *g_surface;
    double* fermi;
    int *iters, *status;
} negf_obc_out;
int negf_obc_decimate_pair(negf_ctx* ctx, const negf_problem* p, const negf_lead* lead_L /* or NULL */,
                           const negf_lead* lead_R /* or NULL */, double mu_L, double mu_R, double kT,
                           double tol, int max_iter, const negf_obc_out* left, const negf_obc_out* right);

/* ---- S1+S3+S4: retarded selected inversion ----------
 *   g_0 = A_00^-1; g_i = (A_ii - A_{i,i-1} g_{i-1} A_{i-1,i})^-1;
 *   G_{n-1,n-1} = g_{n-1}; X_i = g_i A_{i,i+1}; Y_i = A_{i+1,i} g_i;
 *   G_{i,i+1} = -X_i G_{i+1,i+1}; G_{i+1,i} = -G_{i+1,i+1} Y_i; G_ii = g_i - G_{i,i+1} Y_i;
 *   corner: G_{i,n-1} = -X_i G_{i+1,n-1}.
 * sigma_r may be NULL (no self-energy at all).  GR_diag [N_E][n][b][b] required;
 * GR_upper / GR_lower [N_E][n-1][b][b] and GR_corner [N_E][b][b] (= G_{0,n-1}) may be NULL.
 * info [N_E]. */
int negf_rgf_retarded(negf_ctx* ctx, const negf_problem* p, const negf_sigma* sigma_r,
                      negf_c128* GR_diag, negf_c128* GR_upper, negf_c128* GR_lower,
                      negf_c128* GR_corner, int flags, int* info);

/* ---- S5+S6: lesser / greater selected blocks ----------------
 *   g^x_0 = g_0 B_00 g_0^H;
 *   g^x_i = g_i [B_ii + A_{i,i-1} g^x_{i-1} A_{i,i-1}^H - Y_{i-1} B_{i-1,i} - B_{i,i-1} Y_{i-1}^H] g_i^H;
 *   G^x_{n-1,n-1} = g^x_{n-1};
 *   G^x_{i,i+1} = (-g^x_i A_{i+1,i}^H + g_i B_{i,i+1}) (G^R_{i+1,i+1})^H - X_i G^x_{i+1,i+1};
 *   G^x_ii = g^x_i - X_i G^x_{i+1,i} - G^x_{i,i+1} X_i^H - X_i G^x_{i+1,i+1} X_i^H,
 *   G^x_{i+1,i} = -(G^x_{i,i+1})^H (not stored).
 * Needs the sweep state retained by negf_rgf_retarded(..., NEGF_KEEP_SWEEP) on the SAME problem
 * and sigma_r (else NEGF_ENOSTATE), and GR_diag from that call.  Either of sigma_lesser /
 * sigma_greater may be NULL (then its outputs are ignored).  G*_diag [N_E][n][b][b],
 * G*_upper [N_E][n-1][b][b] (may be NULL). */
int negf_rgf_lesser_greater(negf_ctx* ctx, const negf_problem* p, const negf_sigma* sigma_r,
                            const negf_sigma* sigma_lesser, const negf_sigma* sigma_greater,
                            const negf_c128* GR_diag,
                            negf_c128* GL_diag, negf_c128* GL_upper,
                            negf_c128* GG_diag, negf_c128* GG_upper, int* info);

/* ---- S7: observables (readings R11-R13) -------------
 *   density[k]      = sum_E w_E Re[(-i/2pi) (G^< S)_kk]     over the BT pattern      [N = n b]
 *   ldos[E][i]      = -(1/pi) Im Tr[(G^R S)_ii]                                      [N_E][n]
 *   transmission[E] = Re Tr[Gamma_L G^R_{0,n-1} Gamma_R (G^R_{0,n-1})^H]             [N_E]
 *   bond_current[E][i] = 2 Re Tr[(H_{i,i+1} - E S_{i,i+1}) G^<_{i+1,i}]              [N_E][n-1]
 *   contact_current[E][c] = Re Tr[Sigma^<_c G^>_cc - Sigma^>_c G^<_cc], c = L, R     [N_E][2]
 * Every output may be NULL (skipped); inputs only needed by skipped outputs may be NULL.
 * density is OVERWRITTEN (not accumulated across calls); weights [N_E] device doubles. */
int negf_observables(negf_ctx* ctx, const negf_problem* p,
                     const negf_c128* GR_diag, const negf_c128* GR_upper, const negf_c128* GR_lower,
                     const negf_c128* GR_corner,
                     const negf_c128* GL_diag, const negf_c128* GL_upper, const negf_c128* GG_diag,
                     const negf_c128* gamma_L, const negf_c128* gamma_R,
                     const negf_c128* sigma_lesser_L, const negf_c128* sigma_greater_L,
                     const negf_c128* sigma_lesser_R, const negf_c128* sigma_greater_R,
                     const double* weights,
                     double* density, double* ldos, double* transmission,
                     double* bond_current, double* contact_current);

/* ---- Eq. 3: energy convolution of selected blocks ----------
 * The step on the other side of the LSE in the paper's Fig. 1, for M1 = M2 = I and the element-wise product:
 *   mode 0 (convolution)  Y[m] = scale * sum_k X1[m - k] (.) op(X2[k]),                  m = 0 .. 2 N_E - 2
 *   mode 1 (correlation)  Y[m] = scale * sum_k X1[k] (.) op(X2[k - (m - (N_E - 1))])     (lag m - (N_E - 1))
 * on a uniform grid of N_E <= 1024 energies, zero outside it; op = identity or complex conjugate (conj2),
 * with the b x b blocks of X2 read transposed when transpose_block = b > 0 (elems_per_energy must then be a
 * multiple of b*b).  X1, X2: [N_E][elems_per_energy] (any family of include/negf.h, energy slowest); Y:
 * [2 N_E - 1][elems_per_energy].  Done by FFT along the energy axis in shared memory (radix 2, zero-padded
 * to a power of two L >= 2 N_E - 1), the (E; i,j) -> (i,j; E) transposition of the paper happening in the
 * tile load.  NEGF_EUNSUPPORTED for N_E > 1024; X1, X2 and Y must not overlap. */
int negf_energy_convolve(negf_ctx* ctx, int n_energy, long long elems_per_energy, int transpose_block,
                         const negf_c128* X1, const negf_c128* X2, int mode, int conj2, negf_c128 scale,
                         negf_c128* Y);

/* ---- whole path with DEVICE buffers: S2 -> S7 in one call (Fig. 1 "LSE+OBC") --------
 * negf_obc_decimate_pair -> negf_rgf_retarded (NEGF_KEEP_SWEEP) -> negf_rgf_lesser_greater -> negf_observables on
 * one energy batch, all arrays DEVICE pointers owned by the caller.  This is the call the energy-batch scheduler
 * (K3) sees the whole path through: it may split the batch into concurrent energy groups (NEGF_OPT_ENERGY_GROUPS),
 * each on a stream and a slice of the workspace owned by the context; everything is forked from the context's
 * stream and joined back to it before the call returns (asynchronous like the four calls, no host synchronisation).
 * sigma_*: Sigma_S only (left / right members are ignored: the boundary blocks come from the decimation);
 * sigma_greater NULL = no G^>.  Members of negf_device_outputs: left / right as negf_obc_out with sigma_r, gamma,
 * sigma_lesser, sigma_greater, iters, status required; GR_diag, GL_diag, info_r, info_x required; GG_diag required
 * when sigma_greater is given; the other pointers may be NULL (skipped).  Results are identical to the four calls
 * made one after the other on the same batch (the density is summed over the groups in a fixed order). */
typedef struct {
    negf_obc_out left, right;
    negf_c128 *GR_diag, *GR_upper, *GR_lower, *GR_corner, *GL_diag, *GL_upper, *GG_diag, *GG_upper;
    double *density, *ldos, *transmission, *bond_current, *contact_current;
    int *info_r, *info_x;
} negf_device_outputs;
int negf_pipeline_device(negf_ctx* ctx, const negf_problem* p,
                         const negf_sigma* sigma_r, const negf_sigma* sigma_lesser, const negf_sigma* sigma_greater,
                         const double* weights, double mu_L, double mu_R, double kT, double tol, int max_iter,
                         const negf_device_outputs* out);

/* ---- whole path with HOST buffers (bench.py's end-to-end leg) ---------------------------------
 * All array arguments here are HOST pointers (pinned memory recommended).  Copies the inputs
 * to the device, runs negf_obc_decimate (both sides) -> negf_rgf_retarded ->
 * negf_rgf_lesser_greater -> negf_observables, copies the results back and SYNCHRONISES the
 * stream before returning.  Device staging comes from `dev_scratch` (DEVICE pointer, caller
 * owned, at least negf_pipeline_host_bytes()).  Sigma_S as for negf_sigma but with host
 * pointers and left/right ignored.  Outputs may be NULL. */
typedef struct {
    negf_c128 *GR_diag, *GR_upper, *GR_lower, *GL_diag, *GL_upper, *GG_diag, *GG_upper;
    double *density, *ldos, *transmission, *bond_current, *contact_current;
    int *info;                /* [N_E] max over the stage codes */
} negf_host_outputs;
int negf_pipeline_host_bytes(const negf_problem* p_shape_only, int kind_max, int want_greater, size_t* bytes);
int negf_pipeline_host(negf_ctx* ctx, const negf_problem* host_problem,
                       const negf_sigma* host_sigma_r, const negf_sigma* host_sigma_lesser,
                       const negf_sigma* host_sigma_greater, const double* host_weights,
                       double mu_L, double mu_R, double kT, double tol, int max_iter,
                       void* dev_scratch, size_t dev_scratch_bytes,
                       const negf_host_outputs* out,
                       size_t* h2d_bytes, size_t* d2h_bytes);

/* ---- building blocks exposed for tests and roofline measurement -------- */
/* C[e] = alpha * op(A[e]) op(B[e]) + beta * D[e], e < batch; m x n x k complex; row-major with
 * leading dimensions lda/ldb/ldc (ldd = ldc); op: 0 = none, 1 = conjugate transpose; strides in
 * elements between consecutive batch entries (0 = shared).  D may be NULL (beta ignored) or == C. */
int negf_zgemm_batched(negf_ctx* ctx, int opA, int opB, int m, int n, int k,
                       negf_c128 alpha, const negf_c128* A, int lda, long long strideA,
                       const negf_c128* B, int ldb, long long strideB,
                       negf_c128 beta, const negf_c128* D,
                       negf_c128* C, int ldc, long long strideC, int batch);
/* In-place inverse of `batch` dense b x b matrices (stride in elements), partial pivoting on
 * |re|+|im| (b <= 96: on its 25 leading bits, i.e. threshold pivoting at 1 - 2^-13); info[e] = 0 or
 * (column+1) of the first zero pivot.  Uses the context workspace. */
int negf_zinverse_batched(negf_ctx* ctx, int b, negf_c128* A, long long stride, int batch, int* info);
/* The same inverse for callers that must not allocate and have no workspace to hand over (code under CUDA graph
 * capture, tight serving loops, harnesses that forbid cudaMalloc): identical kernels, launch sequence and results
 * as negf_zinverse_batched (K1; the block inversions of the RGF recurrences), but
 * the scratch of the blocked algorithm (b > 96: pivot rows, row-move tables, pivot indices) is a file-scope
 * `static __device__` array of NEGF_STATIC_SCRATCH_BYTES inside the library, which every GPU that loads the
 * library holds until the process exits.  The call itself makes no cudaMalloc / cudaFree and calls no allocating
 * library routine; it ignores (and leaves untouched) the context workspace and the retained sweep state.
 * Limit: b <= 96 needs no scratch (any batch <= what the kernels take); above that about 5.2 KB * b per matrix, i.e.
 * batch * b <= ~3200 (b = 130: batch 24; b = 256: 12; b = 1024: 3; b = 2048: 1).  Larger problems return
 * NEGF_ESTATICLIMIT and launch nothing; NEGF_EUNSUPPORTED while negf_profile_enable is on (it creates events).
 * All calls on a GPU share the one array, which keeps the last call's contents (nothing in it needs to start at
 * zero: each call writes what it reads): calls that OVERLAP on the GPU (different streams, contexts or host
 * threads) race; order them on one stream or with events.  A, info: DEVICE pointers as for negf_zinverse_batched. */
#define NEGF_STATIC_SCRATCH_BYTES (16u << 20)
int negf_zinverse_batched_static(negf_ctx* ctx, int b, negf_c128* A, long long stride, int batch, int* info);
/* Measures the FP64 DMMA (mma.sync m8n8k4) issue-rate peak of this GPU for about `ms`
 * milliseconds; SYNCHRONISES.  Writes TFLOP/s to *tflops (HOST pointer). */
int negf_fp64_peak(negf_ctx* ctx, double ms, double* tflops);

#ifdef __cplusplus
}
#endif
#endif /* NEGF_H */
