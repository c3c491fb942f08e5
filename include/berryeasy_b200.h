/*
 * berryeasy_b200.h -- C ABI of the B200-native Wilson-loop hot path of BerryEasy
 * (A. C. Tyner, arXiv 2312.13051; citations "PAPER.md:<line>" refer to /root/reference/PAPER.md,
 * "R<n>" to the readings listed in DESIGN.md).
 *
 * The library takes an already assembled grid of Bloch / supercell Hamiltonians H(k) and returns
 * Wannier-centre-charge phases.  Every step runs in hand-written sm_100a CUDA kernels; there is
 * no cuSOLVER / cuBLAS inside and no CPU fallback.
 *
 * Common conventions
 * ------------------
 *  - complex128 = interleaved (re, im) pairs of IEEE double, 16-byte aligned.
 *  - A Hamiltonian is a dense row-major [N][N] complex128 array, Hermitian, full storage (only
 *    the upper triangle H[r][c], c >= r, is read).
 *  - H_grid layout: [batch][dims[0]]..[dims[ndim-1]][N][N], last grid axis fastest (be_grid).
 *  - "d" prefixed pointers are DEVICE pointers, "h" prefixed pointers are HOST pointers.
 *  - Ownership: the caller owns every data buffer; the library never frees them and keeps no
 *    reference past the call.  be_ctx owns only scratch memory (allocated lazily with
 *    cudaMallocAsync-free plain cudaMalloc, grown on demand, released by be_destroy).
 *  - Asynchrony: device entry points enqueue all work on the context's stream and return; outputs
 *    are valid once the caller synchronises that stream.  (Scratch growth may synchronise.)
 *    *_host entry points are synchronous: they return after the host outputs are written.
 *  - Errors: return value 0 = BE_OK; negative = argument / shape / alignment error detected on the
 *    host before anything is enqueued; positive = CUDA runtime error (cudaError_t value).
 *    Size limits (BE_ERR_UNSUPPORTED, checked before anything is enqueued): N <= 6400 for every entry
 *    point that diagonalizes H, n_occ (bands of a Wilson matrix) <= 2048.
 *    Numerical trouble is never an error return: be_eigh_batched reports it per matrix in d_info; the
 *    Wilson entry points (be_wilson_loop*, be_spin_resolved_wilson*) have no d_info, so the phases of
 *    every loop (sector) with a flagged eigensolve of H or of the projected spin operator (inverse
 *    iteration / cluster orthogonalization failure, non-finite eigenvalue) or a Wilson matrix whose QR
 *    iteration did not converge come back as NaN -- never as plausible numbers.  d_mingap flags loops
 *    without a spectral gap.
 *  - Devices: a context belongs to the device that was current in be_create; every entry point makes that
 *    device current for its duration and restores the caller's.
 *  - Thread safety: one context per host thread; no global state.
 *  - Phases are returned in radians, ascending, on the branch (-pi, pi] (R7).  The library's
 *    W = prod_j U_j^dagger U_{j+1} is the Hermitian conjugate of the paper's product (Eq. 2,
 *    PAPER.md:38), so the paper's WCC is xbar_n = -theta_n / 2 pi (mod 1) (R3).
 */
#ifndef BERRYEASY_B200_H
#define BERRYEASY_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define BE_OK                 0
#define BE_ERR_NULL          -1   /* required pointer is NULL                                  */
#define BE_ERR_SHAPE         -2   /* N, n_occ, dims, dir ... out of range                      */
#define BE_ERR_ALIGN         -3   /* pointer not 16-byte (complex) / 8-byte (double) aligned   */
#define BE_ERR_UNSUPPORTED   -4   /* valid request this build cannot serve (stated per call)   */
#define BE_ERR_NOMEM         -5   /* scratch allocation failed                                 */
#define BE_ERR_STATIC_LIMIT  -6   /* request exceeds the fixed scratch of a *_static entry     */

typedef struct be_ctx be_ctx;   /* opaque; owns scratch only */

typedef struct {
  int     ndim;      /* number of grid axes after the batch axis, 1..3                          */
  int64_t batch;     /* independent realizations, >= 1                                          */
  int     dims[3];   /* points per grid axis; unused trailing entries ignored                   */
  int     N;         /* orbitals: every H is [N][N]                                             */
} be_grid;

/* Create / destroy a context bound to a CUDA stream (cudaStream_t passed as void*; NULL = the
 * legacy default stream).  The current CUDA device at creation time is used for all scratch. */
int be_create(be_ctx** out, void* cuda_stream);
int be_destroy(be_ctx* ctx);
const char* be_strerror(int code);

/* Upper bound, in bytes, on the scratch one call with these shapes allocates (informative; op:
 * 0 = eigh, 1 = wilson loop, 2 = nested, 3 = spin resolved). */
size_t be_workspace_bytes(const be_grid* grid, int n_occ, int op);

/* Cap on the scratch used for per-chunk work buffers (default: 70 % of the device memory, 134 GB on a
 * B200).  Work is processed in chunks of whole loops sized to stay under the cap and under what the device
 * has free when the call is made (free memory + the scratch the context already holds - 2 GiB). */
int be_set_workspace_limit(be_ctx* ctx, size_t bytes);

/* Two-stream chunk pipeline for be_wilson_loop / be_spin_resolved_wilson when the work is split
 * into several chunks (default OFF).  ON: the tridiagonalization of chunk c+1 (HBM bound) runs on the
 * context's stream while the rest of chunk c (FP64 / latency bound) runs on an internal
 * high-priority stream, with two scratch regions and one GEMM CTA + one k_hemv CTA sharing each SM;
 * the caller's stream is joined before return, so the call's semantics do not change.  Measured on
 * the N = 1600 bench workload it is a wash (3.42 s vs 3.38 s per step: the GEMM kernel loses at one
 * CTA per SM what the overlap gains -- DESIGN.md section 11), hence the default. */
int be_set_chunk_pipeline(be_ctx* ctx, int on);

/* Frees the scratch the context holds (work arena, host-variant staging buffers); it is re-allocated on
 * demand by the next call.  Synchronises the context's streams.  For callers that need the device memory
 * back between calls (the arena of a large call stays allocated otherwise). */
int be_release_workspace(be_ctx* ctx);

/* Algorithm of the Hermitian tridiagonalization inside S1:
 *   0  one-stage blocked Householder reduction (half of its flops are matrix-vector products streamed
 *      from HBM once per column);
 *   1  two-stage reduction: dense -> band of width 8 in ONE fused tensor-core pass over the trailing
 *      matrix per 8 columns, band -> tridiagonal by bulge chasing, eigenvectors back-transformed
 *      through both stages, for every 128 <= N <= 2048;
 *   2  (default) two-stage where it was measured faster (N >= 1024), one-stage below.
 * Outside 128 <= N <= 2048 the setting is ignored (N <= 104: on-chip paths; N > 2048: one-stage).  Both
 * produce eigenpairs to the same tolerance; selectable per context so that they can be timed on the
 * same input.  Returns BE_ERR_SHAPE for any other value. */
int be_set_eigh_algorithm(be_ctx* ctx, int algo);

/* FP64 peak probe (measurement aid for bench.py's roofline, not part of the path): runs a chain of
 * which = 0: DMMA.8x8x4 (mma.sync.m8n8k4.f64), 1: DFMA with reused operands, 2: DFMA with three distinct
 * register operands per instruction, on every SM of the context's device and stream, and writes the
 * achieved rate in TFLOP/s to *tflops (host pointer).  Synchronises the stream; ~20 ms. */
int be_probe_fp64(be_ctx* ctx, int which, double* tflops);

/* Number of kernels launched by this context since creation (for bench.py's gpu_launches). */
int64_t be_launch_count(const be_ctx* ctx);

/* Bytes of H_grid the *_host entry points have copied host -> device since the context was created (bench.py's
 * h2d_bytes_per_step).  Matrices of order >= 256 travel as row blocks of their upper triangle, see the host variants. */
int64_t be_host_grid_bytes_copied(const be_ctx* ctx);

/* How the last be_wilson_loop_host / be_spin_resolved_wilson_host call of this context streamed its grid: n > 0 =
 * n chunks of whole loops, each processed on its own; n < 0 = ONE chunk fed in -n sub-ranges (two-stage eigensolver:
 * only the dense -> band stage runs per sub-range); 0 = no such call yet. */
int be_host_schedule(const be_ctx* ctx);

/* Optional per-kernel-class profile (bench.py's roofline): when enabled every launch of an
 * instrumented kernel class is bracketed by a CUDA event pair on the context's stream and its
 * algorithmic bytes / flops are accumulated.  be_profile_enable resets the counters (it
 * synchronises the stream); be_profile_get synchronises and returns the summed event time in ms.
 * Classes 0..be_profile_name(i)==NULL: "hemv" (k_hemv, or the on-chip
 * tridiagonalization for N <= 104), "colw", "zgemm", "bisect", "invit", "cluster_orth", "hessenberg", "hqr",
 * "jacobi", "misc". */
int be_profile_enable(be_ctx* ctx, int on);
const char* be_profile_name(int cls);
int be_profile_get(be_ctx* ctx, int cls, double* ms, int64_t* launches, double* bytes, double* flops);

/*
 * S1 -- batched Hermitian eigensolve ("exact diagonalization of a discretized
 * Hamiltonian at many points in reciprocal space").
 *   dH     [count][N][N] complex128, Hermitian, not modified.  Only the row-major upper triangle (diagonal
 *          included) is read, here and in every call that takes an H_grid.
 *   dE     [count][N] double: all eigenvalues, ascending.
 *   dU     [count][N][n_vec] complex128, may be NULL: U[c][r][v] = component r of the eigenvector of
 *          the v-th lowest eigenvalue; columns orthonormal.  0 <= n_vec <= N.
 *   d_info [count] int, may be NULL: 0 = converged; >0 = number of vectors whose inverse iteration
 *          or Jacobi sweep limit did not meet its tolerance.
 * Paths: N <= 8 cyclic one-sided Jacobi on the shifted matrix, one thread per matrix; otherwise
 * blocked Householder tridiagonalization + bisection + inverse iteration (clusters of close
 * eigenvalues re-orthogonalized after every solve) + compact-WY back-transform, all matrices of the
 * batch advanced in lock step.  N <= 6400 (shared-memory staging of one column), else
 * BE_ERR_UNSUPPORTED.
 */
int be_eigh_batched(be_ctx* ctx, const void* dH, int64_t count, int N, int n_vec,
                    double* dE, void* dU, int* d_info);

/*
 * S1, variant that allocates nothing: for callers that cannot call cudaMalloc (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid it).  Same arguments, layouts and results as be_eigh_batched on the
 * Jacobi path (N <= 8, else BE_ERR_UNSUPPORTED); the eigenvector frames the kernel writes before they are
 * transposed to dU go to a fixed device array of BE_STATIC_EIGH_MAX_ELEMS complex128 (8 MiB), which every GPU
 * that loads the library holds until the process exits, instead of the context workspace.
 *   Limit: count <= BE_STATIC_EIGH_MAX_ELEMS and count * N * max(n_vec, 1) <= BE_STATIC_EIGH_MAX_ELEMS
 *   (e.g. 32768 matrices of N = 4 with all vectors), else BE_ERR_STATIC_LIMIT; nothing is enqueued then.
 *   No cudaMalloc / cudaFree / allocating routine is called (leave be_profile_enable off: the profile grows its
 *   event pool on demand).  The array is shared by every context of the process on that device and keeps the
 *   last call's contents (each call overwrites the part it reads): two calls that overlap on the GPU (different
 *   streams or contexts without ordering) race on it -- serialize them.  Work is enqueued on the context stream.
 */
#define BE_STATIC_EIGH_MAX_ELEMS ((size_t)1 << 19)
int be_eigh_batched_static(be_ctx* ctx, const void* dH, int64_t count, int N, int n_vec,
                           double* dE, void* dU, int* d_info);

/*
 * S1-S4 -- hybrid Wannier-centre-charge surface (``WSurf``, Eq. 2
 * Eq. 3): for every batch entry and every grid point of the axes other than
 * ``dir`` one discretized, path-ordered Wilson loop along axis ``dir`` over the n_occ lowest bands
 *     W = prod_{j=0}^{N1-1} U_j^dagger U_{j+1},   U_{N1} := diag(Phi) U_0,   theta = arg eig(W).
 * No unitarization of links or of W (R4); exactly N1 = dims[dir] links, all points distinct (R5).
 *   d_close  [N] complex128 unit-modulus Phi_alpha = exp(-i G.r_alpha) (R6), NULL = identity.
 *   d_theta  [loops][n_occ] double, loops = batch * prod(dims other than dir), row-major over
 *            (batch, remaining axes in order); ascending in (-pi, pi].
 *   d_abs    same shape, |lambda_n| in the order of d_theta; may be NULL.
 *   d_mingap [loops] double, min over the loop of E[n_occ]-E[n_occ-1] (+inf if n_occ == N);
 *            a value <= 1e-8 ||H|| marks a loop without a spectral gap (R8); may be NULL.
 */
int be_wilson_loop(be_ctx* ctx, const void* dH_grid, const be_grid* grid, int n_occ, int dir,
                   const void* d_close, double* d_theta, double* d_abs, double* d_mingap);

/*
 * S5 -- nested Wilson loop (``WNWL``, Eq. 8; R9).
 * grid->ndim >= 2.  For every point of axis dir2 (and every batch entry / remaining axis) the loop
 * along dir1 is started at index ``base``; the right eigenvectors of W whose phases rank
 * wb_lo..wb_hi-1 on the branch (theta_cut - 2 pi, theta_cut] span the Wannier-band subspace V_S
 * (orthonormalized); w = U_base V_S; a second loop of w runs along dir2 (closing phase d_close2).
 *   d_theta1       [batch][other][dims[dir2]][n_occ]: first-level phases, branch (-pi, pi].
 *   d_theta_nested [batch][other][wb_hi-wb_lo]: nested phases; polarization p = -sum/2pi mod 1.
 * n_occ <= 2: closed-form eigenvectors of the 2 x 2 Wilson matrix (the paper's 4-band quadrupole
 * models, BASELINE.json configs[1]).  n_occ > 2: all eigenvalues of W by Hessenberg-QR, the selected
 * ones refined to eigenvectors by inverse iteration on W - lambda I (partially pivoted LU per band,
 * every solve followed by the orthonormalization, so degenerate Wannier bands span their cluster);
 * wb_hi - wb_lo <= 64, else BE_ERR_UNSUPPORTED.  The result is defined when the selected bands are
 * separated from the others by a Wannier gap (R9).
 */
int be_nested_wilson(be_ctx* ctx, const void* dH_grid, const be_grid* grid, int n_occ,
                     int dir1, int dir2, int base, int wb_lo, int wb_hi, double theta_cut,
                     const void* d_close1, const void* d_close2,
                     double* d_theta1, double* d_theta_nested);

/*
 * band windows (``bands``, "the list of band indices"): the loop
 * of the bands [band_lo, band_hi) in ascending-energy order instead of the lowest n_occ (band_lo = 0,
 * band_hi = n_occ is be_wilson_loop).  The lowest band_hi eigenvectors are computed at every k and the
 * window's columns are looped; outputs have m = band_hi - band_lo columns.
 *   d_mingap [loops]: min over the loop of the gaps at BOTH edges of the window, E[band_lo]-E[band_lo-1]
 *            (band_lo > 0) and E[band_hi]-E[band_hi-1] (band_hi < N); +inf without an inner edge.
 * 0 <= band_lo < band_hi <= N, else BE_ERR_SHAPE.  All other arguments as in be_wilson_loop /
 * be_spin_resolved_wilson (m_lo = -1 means m / 2; d_pso [loops][N1][m]).
 */
int be_wilson_loop_window(be_ctx* ctx, const void* dH_grid, const be_grid* grid, int band_lo, int band_hi,
                          int dir, const void* d_close, double* d_theta, double* d_abs, double* d_mingap);
int be_spin_resolved_wilson_window(be_ctx* ctx, const void* dH_grid, const be_grid* grid, int band_lo,
                                   int band_hi, int dir, const void* dS, int S_is_diag, int m_lo,
                                   const void* d_close, double* d_theta_lo, double* d_theta_hi, double* d_pso);

/*
 * S6 -- spin-resolved Wilson loop (``WSpinSurf``): at every k the reduced
 * projected spin operator U^dagger S U (the non-zero block of P S P) is
 * diagonalized, S_red = V Sigma V^dagger (ascending); the occupied frame is rotated into the
 * lower sector U V[:, :m_lo] and the upper sector U V[:, m_lo:] and each sector is looped (R10).
 *   dS         S_is_diag = 1: [N] double (real diagonal);  0: [N][N] complex128 row-major.
 *   m_lo       size of the lower sector; -1 = n_occ / 2.
 *   d_theta_lo [loops][m_lo], d_theta_hi [loops][n_occ-m_lo] (either may be NULL).
 *   d_pso      [loops][N1][n_occ] PSO eigenvalues ascending (``spin_spectrum``);
 *              may be NULL.
 */
int be_spin_resolved_wilson(be_ctx* ctx, const void* dH_grid, const be_grid* grid, int n_occ,
                            int dir, const void* dS, int S_is_diag, int m_lo, const void* d_close,
                            double* d_theta_lo, double* d_theta_hi, double* d_pso);

/*
 * S2/S3 building block -- batched complex128 GEMM on the FP64 tensor cores (DMMA), column-major:
 *     C[b] = alpha * op(A[b]) * op(B[b]) + beta * C[b],   b = 0..batch-1,  X[b] = X + b * strideX
 * op: 0 = N, 1 = T, 2 = C (conjugate transpose), 3 = J (conjugate).  Supported pairs: NN, NC, CN, NT,
 * TN, JN, NJ, CC, TJ (others: BE_ERR_UNSUPPORTED).  This is the contraction behind the link overlaps
 * M_j = U_j^dagger U_{j+1} (op C,N) and the ordered product (op N,N).
 * alpha, beta: pointers to 2 doubles (re, im) on the HOST.  lower != 0: only tiles on or below the
 * diagonal are computed.  All matrix pointers are device pointers, strides in complex elements.
 */
int be_zgemm_batched(be_ctx* ctx, int opA, int opB, int M, int N, int K,
                     const double* alpha, const void* dA, int lda, int64_t strideA,
                     const void* dB, int ldb, int64_t strideB,
                     const double* beta, void* dC, int ldc, int64_t strideC, int64_t batch, int lower);

/*
 * S7 -- winding of Theta_i = sum_n theta_n over a closed transverse cycle (Eq. 6):
 *   d_theta [n_cycles][n_points][m]  ->  d_wind [n_cycles] double,
 *   wind = (1/2pi) sum_i wrap(Theta_{i+1} - Theta_i), indices cyclic.  Paper's C = -wind (R3).
 */
int be_winding(be_ctx* ctx, const double* d_theta, int64_t n_cycles, int n_points, int m,
               double* d_wind);

/*
 * Step before the path (the Bloch / supercell Hamiltonian at a
 * wave vector, with boundary phases, is what the paper gets from PyBinding): H_grid assembled on the
 * device from real-space blocks,
 *     H[k] = sum_R coef[k][R] * A[R],     coef[k][R] = exp(2 pi i  t_k . R)   (t = reduced coordinates),
 * as ONE complex GEMM (N^2 x nR) x (nR x count) on the FP64 tensor cores.
 *   be_bloch_coefficients: d_t [count][nd] double reduced coordinates (nd = 1..3), h_R [nR][nd] int
 *          lattice vectors on the HOST, d_coef [count][nR] complex128 out.
 *   be_assemble_bloch: dA [nR][N][N] complex128 row-major blocks (the caller lists A_R and, for R != 0,
 *          A_{-R} = A_R^dagger explicitly; twisted boundaries: the blocks of the wrapping hops with
 *          R = +-e_x, +-e_y), d_coef as above (any complex coefficients are accepted), dH [count][N][N]
 *          out.  Hermiticity of the result is the caller's (the blocks') responsibility.
 */
int be_bloch_coefficients(be_ctx* ctx, const double* d_t, const int* h_R, int nd, int nR, int64_t count,
                          void* d_coef);
int be_assemble_bloch(be_ctx* ctx, const void* dA, const void* d_coef, int64_t count, int N, int nR, void* dH);

/*
 * The same step FUSED in front of S1: be_wilson_loop / be_spin_resolved_wilson on a grid that is never
 * materialised.  H at grid point (i_0, .., i_{ndim-1}) of batch entry b is
 *     H = sum_R exp(2 pi i sum_a (i_a / dims[a]) R[a]) * A[b][R],
 * generated chunk by chunk straight into the eigensolver's work copy (no 17-43 GB H_grid, no read of it).
 *   dA  [batch][nR][N][N] complex128 row-major blocks (every batch entry -- disorder realization -- has
 *       its own set; list A_R and A_{-R} = A_R^dagger both), h_R [nR][ndim] int lattice vectors on the HOST.
 * All other arguments, outputs and conventions as in be_wilson_loop / be_spin_resolved_wilson.
 */
int be_wilson_loop_bloch(be_ctx* ctx, const void* dA, const int* h_R, int nR, const be_grid* grid, int n_occ,
                         int dir, const void* d_close, double* d_theta, double* d_abs, double* d_mingap);
int be_spin_resolved_wilson_bloch(be_ctx* ctx, const void* dA, const int* h_R, int nR, const be_grid* grid,
                                  int n_occ, int dir, const void* dS, int S_is_diag, int m_lo, const void* d_close,
                                  double* d_theta_lo, double* d_theta_hi, double* d_pso);

/*
 * Plaquette mode ("integrated Berry flux through one plaquette",
 * the coupling-matrix method and its spin-resolved generalization): on a periodic 2D grid
 * (grid->ndim == 2, dims = (ny, nx)) every point is diagonalized ONCE and
 *     flux[j][i] = arg det( L_x(j,i) L_y(j,i+1) L_x(j+1,i)^dagger L_y(j,i)^dagger )  in (-pi, pi],
 *     L_x(j,i) = U(j,i)^dagger U(j,i+1),  L_y(j,i) = U(j,i)^dagger U(j+1,i)   (indices cyclic, R4: no
 * unitarization; the determinant by partially pivoted LU).  sum(flux) / 2 pi is the Chern number in the
 * orientation of the paper's Eq. 6 flow (Eq. 4: +1).
 *   dS NULL: d_flux [batch][ny][nx] of the n_occ lowest bands; d_flux_hi, d_pso ignored.
 *   dS given (S_is_diag / m_lo as in be_spin_resolved_wilson): d_flux = lower PSO sector, d_flux_hi =
 *   upper sector (may be NULL), d_pso [batch][ny][nx][n_occ] (may be NULL).
 * The whole grid has to fit the workspace cap (be_set_workspace_limit), else BE_ERR_UNSUPPORTED.
 */
int be_plaquette_flux(be_ctx* ctx, const void* dH_grid, const be_grid* grid, int n_occ, const void* dS,
                      int S_is_diag, int m_lo, double* d_flux, double* d_flux_hi, double* d_pso);

/*
 * Host-buffer variants (end-to-end path): h* pointers are host memory (pinned recommended).  The
 * grid is streamed to the device in chunks of whole loops, overlapped with compute on an internal
 * copy stream; results are copied back before return.  Schedule (be_host_schedule reports it):
 *   - two-stage eigensolver (N >= 1024, default algorithm) and workspace for all loops at once: ONE chunk, fed in
 *     three sub-ranges of loops (24 loops of N = 1600: 3 + 7 + 14); only the first stage of the eigensolver runs per
 *     sub-range, while the next one travels; everything else runs over the whole batch;
 *   - else N >= 800: TWO chunks, the first just long enough to hide the copy of the second;
 *   - smaller matrices: growing chunks (1/8 of the loops, 1/4, ... or multiples of a wave of SMs),
 *   so that only the first, small copy is exposed.  Semantics as the device calls above; any loop direction.
 *   The default workspace cap is 85 % of the device memory here (the grid is not device resident); a cap set
 *   with be_set_workspace_limit stands.
 *   Which bytes travel: H(k) is Hermitian and the eigensolver reads only its row-major UPPER triangle
 *   (diagonal included; the other triangle may hold anything, on the host and on the device).  For
 *   N >= 256 each matrix is copied as 8 row blocks, block b with the columns from its first row on: 56 % of
 *   the bytes.  Smaller matrices are copied whole (dir == ndim-1: one contiguous copy per chunk, else one
 *   strided copy per loop).  be_host_grid_bytes_copied counts what was copied.
 * The two staging buffers are kept in the context between calls.  be_nested_wilson_host
 * copies the whole grid in one piece (both levels need the whole plane).
 */
int be_wilson_loop_host(be_ctx* ctx, const void* hH_grid, const be_grid* grid, int n_occ, int dir,
                        const void* h_close, double* h_theta, double* h_abs, double* h_mingap);
int be_spin_resolved_wilson_host(be_ctx* ctx, const void* hH_grid, const be_grid* grid, int n_occ,
                                 int dir, const void* hS, int S_is_diag, int m_lo,
                                 const void* h_close, double* h_theta_lo, double* h_theta_hi,
                                 double* h_pso);
int be_nested_wilson_host(be_ctx* ctx, const void* hH_grid, const be_grid* grid, int n_occ, int dir1, int dir2,
                          int base, int wb_lo, int wb_hi, double theta_cut, const void* h_close1,
                          const void* h_close2, double* h_theta1, double* h_theta_nested);

#ifdef __cplusplus
}
#endif
#endif /* BERRYEASY_B200_H */
