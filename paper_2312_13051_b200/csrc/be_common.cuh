// Shared declarations of the CUDA path: context, launch bookkeeping, complex helpers, the batched
// ZGEMM interface and the internal stage entry points.  Nothing in here is used by oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include <math.h>
#include "../../include/berryeasy_b200.h"

typedef double2 cplx;

__host__ __device__ __forceinline__ cplx mkc(double r, double i) { cplx z; z.x = r; z.y = i; return z; }
__host__ __device__ __forceinline__ cplx cadd(cplx a, cplx b) { return mkc(a.x + b.x, a.y + b.y); }
__host__ __device__ __forceinline__ cplx csub(cplx a, cplx b) { return mkc(a.x - b.x, a.y - b.y); }
__host__ __device__ __forceinline__ cplx cmul(cplx a, cplx b) { return mkc(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
// conj(a) * b
__host__ __device__ __forceinline__ cplx cmulc(cplx a, cplx b) { return mkc(a.x * b.x + a.y * b.y, a.x * b.y - a.y * b.x); }
__host__ __device__ __forceinline__ cplx cconj(cplx a) { return mkc(a.x, -a.y); }
__host__ __device__ __forceinline__ cplx cscale(double s, cplx a) { return mkc(s * a.x, s * a.y); }
__host__ __device__ __forceinline__ double cabs2(cplx a) { return a.x * a.x + a.y * a.y; }
__device__ __forceinline__ double cabs1(cplx a) { return fabs(a.x) + fabs(a.y); }
__device__ __forceinline__ cplx cdiv(cplx a, cplx b) {
  // Smith's algorithm
  if (fabs(b.x) >= fabs(b.y)) {
    double r = b.y / b.x, den = b.x + b.y * r;
    return mkc((a.x + a.y * r) / den, (a.y - a.x * r) / den);
  } else {
    double r = b.x / b.y, den = b.x * r + b.y;
    return mkc((a.x * r + a.y) / den, (a.y * r - a.x) / den);
  }
}
// acc += a*b
__device__ __forceinline__ void cfma(cplx& acc, cplx a, cplx b) {
  acc.x = fma(a.x, b.x, acc.x); acc.x = fma(-a.y, b.y, acc.x);
  acc.y = fma(a.x, b.y, acc.y); acc.y = fma(a.y, b.x, acc.y);
}
// acc += conj(a)*b
__device__ __forceinline__ void cfmac(cplx& acc, cplx a, cplx b) {
  acc.x = fma(a.x, b.x, acc.x); acc.x = fma(a.y, b.y, acc.x);
  acc.y = fma(a.x, b.y, acc.y); acc.y = fma(-a.y, b.x, acc.y);
}
// acc -= a*b
__device__ __forceinline__ void cfms(cplx& acc, cplx a, cplx b) {
  acc.x = fma(-a.x, b.x, acc.x); acc.x = fma(a.y, b.y, acc.x);
  acc.y = fma(-a.x, b.y, acc.y); acc.y = fma(-a.y, b.x, acc.y);
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ cplx warp_sum(cplx v) { return mkc(warp_sum(v.x), warp_sum(v.y)); }

// Block-wide sum (all threads get the result).  ``red`` : shared scratch of >= 33 entries of T.
template <typename T>
__device__ __forceinline__ T block_sum(T v, T* red) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
  v = warp_sum(v);
  __syncthreads();
  if (lane == 0) red[w] = v;
  __syncthreads();
  if (w == 0) {
    T t = (lane < nw) ? red[lane] : T{};
    t = warp_sum(t);
    if (lane == 0) red[32] = t;
  }
  __syncthreads();
  return red[32];
}

// ---------------------------------------------------------------------------------------------
struct HostFeed;
struct be_ctx {
  cudaStream_t stream;
  cudaStream_t copy_stream;   // host variants only
  int device;
  int sm_count;
  size_t ws_limit;
  int64_t launches;
  HostFeed* feed;             // consumed (and cleared) by the next large eigensolve
  int host_schedule;          // last *_host call: number of chunks, or -(number of sub-ranges) of the one fed chunk
  int64_t h2d_bytes;          // host -> device bytes of H_grid copied by the *_host entry points since creation
  // scratch arena (bump allocated per call, grown on demand)
  char* arena;
  size_t arena_bytes;
  size_t arena_used;
  int gemm_attr_set;
  // two-stream chunk pipeline (be_wilson_loop / be_spin_resolved_wilson with more than one chunk):
  // the tridiagonalization of chunk c+1 (HBM bound) runs on ``stream`` while everything else of
  // chunk c (FP64 / latency bound) runs on the high-priority ``stream2``
  cudaStream_t stream2;
  cudaEvent_t ev_split, ev_region[2], ev_join;
  int* dR_buf; size_t dR_cap;      // device copy of the lattice vectors of a *_bloch call
  const struct BlochSrc* bloch;   // set while the H eigensolve of a *_bloch call runs: H(k) is assembled, not read
  int chunk_pipeline;         // be_set_chunk_pipeline (default 0)
  int band_lo;                // band window [band_lo, band_lo + m) of the running Wilson call (0 = lowest m bands)
  cudaStream_t side_stream;   // k_q2: the grid of narrow CTAs runs here, next to the grid of full slabs
  cudaEvent_t ev_side[2];
  int split_after_tridiag;    // consumed by be_eigh_large: switch to stream2 after S1a
  int gemm_pad;               // zgemm launches with padded shared memory: at most one GEMM CTA per SM,
                              // leaving room for one k_hemv CTA of the other stream
  struct be_prof* prof;       // optional per-kernel-class CUDA-event timing (be_profile_enable)
  void* stage_buf[2];         // host variants: device staging buffers, kept between calls
  size_t stage_cap[2];        // bytes of each (a two-chunk schedule needs a small and a large one)
  size_t total_mem;           // totalGlobalMem of the device
  int ws_user;                // be_set_workspace_limit was called: the cap is the caller's, not the default
  int invit_solves;           // inverse-iteration solves per eigenvector: 3 (eigenvectors, be_eigh_batched) or 2 (Wilson paths: only the span matters)
  int eigh_algo;              // be_set_eigh_algorithm: 0 one-stage tridiagonalization, 1 two-stage (band) where supported
};

// kernel classes of the profile
enum { PK_HEMV = 0, PK_COL, PK_GEMM, PK_BISECT, PK_INVIT, PK_ORTH, PK_HESS, PK_HQR, PK_JACOBI,
       PK_MISC, PK_FUSED, PK_PANEL, PK_CHASE, PK_Q2, PK_COUNT };
void be_prof_begin(be_ctx* ctx, int cls);
void be_prof_end(be_ctx* ctx, int cls, double bytes, double flops);

// Every extern "C" entry point makes the context's device current for its duration (the scratch arena, the
// internal streams and the function attributes belong to that device) and restores the caller's on return.
struct be_device_guard {
  int prev = -1;
  explicit be_device_guard(const be_ctx* ctx) {
    if (ctx && cudaGetDevice(&prev) == cudaSuccess && prev != ctx->device) cudaSetDevice(ctx->device); else prev = -1;
  }
  ~be_device_guard() { if (prev >= 0) cudaSetDevice(prev); }
};
#define BE_DEVICE_GUARD(ctx) be_device_guard be_guard__(ctx)

// The Wilson-loop paths use the eigenvectors only through the subspaces they span (the occupied space, the PSO
// sectors; W changes by a similarity under a change of basis at a k-point), so the third
// inverse-iteration solve, which only sharpens the individual vectors inside a cluster, is dropped there: after
// TWO solves (each followed by the cluster orthogonalization) the basis is orthonormal to 2e-13 and lies in the
// occupied space to 5e-15, the same as after three (N = 400 supercell, 132 matrices; ONE solve from the random
// start leaves 8e-9 / 3e-11, not enough for |lambda(W)| to 1e-9).  be_eigh_batched, which returns eigenvectors,
// keeps three solves (subspace iteration inside clusters).
struct be_subspace_guard {
  be_ctx* c; int prev;
  explicit be_subspace_guard(be_ctx* ctx) : c(ctx), prev(ctx->invit_solves) { ctx->invit_solves = 2; }
  ~be_subspace_guard() { c->invit_solves = prev; }
};

#define BE_CUDA(x) do { cudaError_t e__ = (x); if (e__ != cudaSuccess) return (int)e__; } while (0)
#define BE_TRY(x) do { int r__ = (x); if (r__ != BE_OK) return r__; } while (0)

// bump allocator on the context arena; pointers stay valid until arena_reset
int  be_arena_reserve(be_ctx* ctx, size_t bytes);   // ensure capacity (may sync + realloc); resets
void* be_arena_alloc(be_ctx* ctx, size_t bytes);
size_t be_effective_ws_limit(be_ctx* ctx, size_t want, bool host_grid = false);   // min(configured cap, what the device can give now); want = the uncapped request    // 256-byte aligned; NULL when exhausted
static inline size_t be_align256(size_t b) { return (b + 255) & ~(size_t)255; }

// ---------------------------------------------------------------------------------------------
// Batched complex GEMM on the FP64 tensor cores (DMMA.8x8x4), column-major operands:
//   C[b] = alpha * op(A[b]) * op(B[b]) + beta * C[b]
// op: 0 = N, 1 = T (transpose), 2 = C (conjugate transpose), 3 = J (conjugate, no transpose).
// Batch b = o * inner + i;  X[b] = X + o * sXo + i * sXi (element strides).
enum { BE_OP_N = 0, BE_OP_T = 1, BE_OP_C = 2, BE_OP_J = 3 };
struct ZgemmParams {
  int M, N, K;
  const cplx* A; int lda; int64_t sAi, sAo;
  const cplx* B; int ldb; int64_t sBi, sBo;
  cplx* C; int ldc; int64_t sCi, sCo;
  int inner; int64_t batch;
  int ringB;          // B uses inner index (i + 1) % inner (next frame of the loop)
  const cplx* phiB;   // with ringB: when i == phi_at, B(k, n) is multiplied by phiB[k] (opB = N)
  int phi_at;         // inner index of the link that crosses the zone boundary (default inner-1)
  cplx alpha, beta;
  int lower;          // 1: skip tiles strictly above the diagonal (C lower triangle, tile granular)
  // optional second K segment: for k >= ksplit the operands are read from A2 / B2 at k - ksplit (same
  // leading dimensions, own outer strides); ksplit = 0: single segment.  Used by the rank-2k update
  // A22 -= [V W] [W V]^H without packing the panels.
  const cplx* A2; const cplx* B2; int64_t sA2o, sB2o; int ksplit;
};
int be_zgemm(be_ctx* ctx, int opA, int opB, const ZgemmParams& p);
static inline ZgemmParams zgemm_simple(int M, int N, int K, const cplx* A, int lda, int64_t sA,
                                       const cplx* B, int ldb, int64_t sB, cplx* C, int ldc,
                                       int64_t sC, int64_t batch) {
  ZgemmParams p;
  p.M = M; p.N = N; p.K = K;
  p.A = A; p.lda = lda; p.sAi = 0; p.sAo = sA;
  p.B = B; p.ldb = ldb; p.sBi = 0; p.sBo = sB;
  p.C = C; p.ldc = ldc; p.sCi = 0; p.sCo = sC;
  p.inner = 1; p.batch = batch;
  p.ringB = 0; p.phiB = nullptr; p.phi_at = -1;
  p.alpha = mkc(1.0, 0.0); p.beta = mkc(0.0, 0.0); p.lower = 0;
  p.A2 = nullptr; p.B2 = nullptr; p.sA2o = p.sB2o = 0; p.ksplit = 0;
  return p;
}

// ---------------------------------------------------------------------------------------------
// Mapping (loop, j) -> matrix index inside H_grid for a loop direction ``dir`` (units: matrices).
struct GridMap {
  int ndim, dir, n1;
  int shift;           // loop point j reads grid index (j + shift) % n1 along dir (nested: base)
  int dims[3];
  int64_t stride[3];
  int64_t batch_stride;
  int64_t loops;       // batch * prod(dims other than dir)
};
__host__ __device__ inline int64_t gridmap_index(const GridMap& g, int64_t loop, int j) {
  int64_t idx = loop, off = 0;
  for (int a = g.ndim - 1; a >= 0; --a) {
    if (a == g.dir) continue;
    int64_t i = idx % g.dims[a];
    idx /= g.dims[a];
    off += i * g.stride[a];
  }
  int jj = j + g.shift; if (jj >= g.n1) jj -= g.n1;
  return off + idx * g.batch_stride + (int64_t)jj * g.stride[g.dir];
}

// ---------------------------------------------------------------------------------------------
// H(k) generated on the fly (be_*_bloch): H[k] = sum_R exp(2 pi i t_k . R) A_R, t = grid index / dims.
struct BlochSrc {
  const cplx* A;        // [batch][nR][N][N]
  const int* dR;        // device [nR][ndim]
  int nR;
  GridMap map;          // decodes (loop, j) into grid indices (the same enumeration as H_grid)
  int64_t loops_per_batch;
};
// matrices c = 0..cnt-1 of the chunk starting at loop0, written to out [cnt][N][N]; coef: scratch [cnt][nR]
int be_bloch_assemble_chunk(be_ctx* ctx, const BlochSrc* bs, int64_t loop0, int64_t cnt, int N, cplx* out);

// Host-resident H_grid streamed chunk by chunk (be_*_host): two device staging buffers filled on the
// copy stream while the previous chunk computes.  Loops must be contiguous (dir == last axis).
// Host grid streamed INTO one chunk (two-stage eigensolver): the matrices arrive in nsub sub-ranges through two
// staging buffers; be_eigh_large gathers each as its copy lands and runs stage 1 (dense -> band) on it while the
// next one travels, then everything else over the whole batch.  issue(self, j) enqueues the copy of sub-range j.
struct HostFeed {
  int nsub;
  int64_t mstart[9];            // matrix index where sub-range j starts (nsub + 1 entries)
  void* buf[2];
  cudaEvent_t copied[2], freed[2];
  int (*issue)(void* self, int j);
  void* self;
};

struct HostStage {
  const char* hH;          // host grid
  size_t loop_bytes;       // n1 * N * N * 16
  size_t mat_bytes;        // N * N * 16
  GridMap hmap;            // (loop, j) -> matrix index inside the host grid (any loop direction)
  void* stage[2];          // device staging buffers (cached in the context), the largest chunk each
  cudaEvent_t copied[2], freed[2];
};
int be_wilson_host_device(be_ctx* ctx, HostStage* hs, const be_grid* grid, int dir, int m, const void* d_close,
                          double* d_theta, double* d_abs, double* d_mingap, const void* dS, int S_is_diag, int m_lo,
                          double* d_theta_lo, double* d_theta_hi, double* d_pso, int spin);

// Stage entry points (host functions enqueueing kernels on ctx->stream)

// Frames-producing eigensolve for ``cnt`` matrices gathered from H via (loop0.., map):
//   matrix c = (loop0 + c / map.n1, c % map.n1).  Outputs:
//   E [cnt][N] ascending;  X [cnt][nv][N] column-major frames (X[c][v*N + r] = U[r][v]);
//   info [cnt] or NULL.  Scratch comes from the context arena (caller reserved it).
//   ne: only E[c][0..ne-1] are computed (ne >= nv; N = all); the rest of the row is left untouched.
int be_eigh_frames(be_ctx* ctx, const cplx* H, const GridMap& map, int64_t loop0, int64_t cnt,
                   int N, int nv, int ne, double* E, cplx* X, int* info);
size_t be_eigh_scratch_bytes(int64_t cnt, int N, int nv);

// eigenphases of ``cnt`` general complex m x m matrices W (column-major, stride m*m, destroyed):
//   theta [cnt][m] ascending in (-pi, pi], absl [cnt][m] or NULL.
int be_eigenphases(be_ctx* ctx, cplx* W, int64_t cnt, int m, double* theta, double* absl, const int* bad = nullptr);
size_t be_eigenphases_scratch_bytes(int64_t cnt, int m);
int be_eigenvalues_general(be_ctx* ctx, cplx* W, int64_t cnt, int m, cplx* lam, int* fail);
int be_sort_phases(be_ctx* ctx, const cplx* lam, int64_t cnt, int m, double* theta, double* absl);
int be_det_phase(be_ctx* ctx, const cplx* W, int64_t cnt, int m, double* phase);
size_t be_nested_general_scratch_bytes(int64_t nl, int m, int ns);
int be_nested_select_general(be_ctx* ctx, cplx* W, int64_t nl, int m, int wb_lo, int wb_hi, double cut,
                             double* theta1, cplx* Vs);

// fused tiny-N loop (small_loop.cu): N <= 8, m <= 2; plain (theta / abs / mingap / W / first frame) or spin resolved
bool be_small_loop_applies(int N, int m, int n1);
int be_small_loop(be_ctx* ctx, const cplx* H, const cplx* frames, const GridMap& map, int N, int m, const cplx* d_close, int phi_at,
                  double* d_theta, double* d_abs, double* d_mingap, cplx* Wout, cplx* X0, const void* dS, int S_is_diag,
                  int m_lo, double* d_theta_lo, double* d_theta_hi, double* d_pso);
int be_eigh_small(be_ctx* ctx, const cplx* H, const GridMap& map, int64_t loop0, int64_t cnt, int N,
                  int nv, double* E, cplx* X, int* info);
int be_eigh_large(be_ctx* ctx, const cplx* H, const GridMap& map, int64_t loop0, int64_t cnt, int N,
                  int nv, int ne, double* E, cplx* X, int* info);
size_t be_eigh_large_scratch_bytes(int64_t cnt, int N, int nv);
// two-stage reduction (eigh_band.cu): dense -> band of width BE_BAND_KB -> tridiagonal
constexpr int BE_BAND_KB = 8;
constexpr int BE_BAND_MINN = 128, BE_BAND_MAXN = 2048, BE_BAND_AUTON = 1024;
size_t be_band_scratch_bytes(int64_t cnt, int N);
int be_band_reduce(be_ctx* ctx, cplx* Bw, int64_t cnt, int N, double* d, double* e, cplx* tau, void* scratch);
int be_band_stage1(be_ctx* ctx, cplx* Bw, int64_t cnt, int N, cplx* tau, void* scratch);
int be_band_stage2(be_ctx* ctx, cplx* Bw, int64_t cnt, int N, double* d, double* e, void* scratch);
int be_band_q2(be_ctx* ctx, const cplx* Bw, cplx* X, int64_t cnt, int N, int nv);
constexpr int BE_MAX_N = 6400;   // largest matrix order of the blocked eigensolver (be_eigh_batched, every Wilson entry point)
constexpr int BE_MAX_M = 2048;   // largest Wilson matrix (bands per sector) of the eigenphase solve
constexpr int TS_MAXN = 104;   // largest matrix reduced entirely in shared memory (tridiag_small.cu)
int be_tridiag_small(be_ctx* ctx, const cplx* H, const GridMap& map, int64_t loop0, int64_t cnt, int N, cplx* Bw,
                     double* d, double* e, cplx* tau, int p0 = 0);
int be_backtransform_small(be_ctx* ctx, const cplx* Bw, const cplx* tau, const double* Z, cplx* X, int64_t cnt, int N,
                           int nv);
size_t be_cluster_orth_scratch_bytes(int64_t cnt, int N, int nv);
int be_cluster_orth(be_ctx* ctx, const double* lam, const double* tnorm, const int* blk, double* Z, int64_t cnt, int N,
                    int nv, double ctol, int* info, void* scratch, int find, int rounds);
int be_frames_to_public(be_ctx* ctx, const cplx* X, cplx* U, int64_t cnt, int N, int nv);
