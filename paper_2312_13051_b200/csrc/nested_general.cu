// S5 for n_occ > 2 -- Wannier-band vectors of the (non-Hermitian, R4) first-level Wilson matrix W:
// the right eigenvectors of the eigenvalues ranked wb_lo..wb_hi-1 on the branch (cut - 2 pi, cut]
// (R9), by inverse iteration on W - lambda I with a partially pivoted LU, orthonormalized per loop
// (only their span enters w = U_base V_S; Eq. 8).  One CTA per (loop, band).
#include "be_common.cuh"
#include <float.h>

namespace {

__device__ __forceinline__ double hash_u(uint64_t x) {
  x += 0x9E3779B97F4A7C15ull; x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull;
  x = (x ^ (x >> 27)) * 0x94D049BB133111EBull; x ^= x >> 31;
  return (double)(x >> 11) * (2.0 / 9007199254740992.0) - 1.0;
}

// lamS [loop][ns]: eigenvalues whose branch angle ranks wb_lo .. wb_hi-1 (ties by index)
__global__ void k_select_bands(const cplx* __restrict__ lam, int m, int wb_lo, int ns, double cut,
                               cplx* __restrict__ lamS) {
  extern __shared__ double th[];
  const int64_t c = blockIdx.x;
  const cplx* l = lam + c * m;
  for (int i = threadIdx.x; i < m; i += blockDim.x) {
    double t = atan2(l[i].y, l[i].x);
    if (t > cut) t -= 2.0 * M_PI;
    if (t <= cut - 2.0 * M_PI) t += 2.0 * M_PI;
    th[i] = t;
  }
  __syncthreads();
  for (int i = threadIdx.x; i < m; i += blockDim.x) {
    const double t = th[i];
    int rank = 0;
    for (int j = 0; j < m; ++j) rank += (th[j] < t) || (th[j] == t && j < i);
    if (rank >= wb_lo && rank < wb_lo + ns) lamS[c * ns + (rank - wb_lo)] = l[i];
  }
}

// A = W - lambda I, PA = LU in place (column-major, unit lower L below the diagonal), piv[k] = row
// swapped with k.  Tiny pivots are replaced by eps ||W||_max (the shift IS an eigenvalue).
__global__ void __launch_bounds__(256) k_lu_shifted(const cplx* __restrict__ W, const cplx* __restrict__ lamS, int m,
                                                    int ns, cplx* __restrict__ LU, int* __restrict__ piv) {
  __shared__ double rv[256];
  __shared__ int ri[256];
  __shared__ double s_scale;
  const int64_t b = blockIdx.x;            // loop * ns + band
  const int64_t c = b / ns;
  const cplx* w = W + c * (int64_t)m * m;
  cplx* A = LU + b * (int64_t)m * m;
  int* pv = piv + b * (int64_t)m;
  const cplx lam = lamS[b];
  const int tid = threadIdx.x;
  double mx = 0.0;
  for (int idx = tid; idx < m * m; idx += 256) {
    cplx a = w[idx];
    mx = fmax(mx, cabs1(a));
    if (idx % m == idx / m) a = csub(a, lam);
    A[idx] = a;
  }
  rv[tid] = mx;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) { if (tid < o) rv[tid] = fmax(rv[tid], rv[tid + o]); __syncthreads(); }
  if (tid == 0) s_scale = fmax(rv[0], DBL_MIN);
  __syncthreads();
  const double tiny = DBL_EPSILON * s_scale;
  for (int k = 0; k < m; ++k) {
    // pivot search in column k
    double best = -1.0; int bi = k;
    for (int i = k + tid; i < m; i += 256) { const double v = cabs1(A[i + (int64_t)k * m]); if (v > best) { best = v; bi = i; } }
    rv[tid] = best; ri[tid] = bi;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
      if (tid < o && (rv[tid + o] > rv[tid] || (rv[tid + o] == rv[tid] && ri[tid + o] < ri[tid]))) { rv[tid] = rv[tid + o]; ri[tid] = ri[tid + o]; }
      __syncthreads();
    }
    const int p = ri[0];
    if (tid == 0) pv[k] = p;
    if (p != k)
      for (int j = tid; j < m; j += 256) { const cplx t = A[k + (int64_t)j * m]; A[k + (int64_t)j * m] = A[p + (int64_t)j * m]; A[p + (int64_t)j * m] = t; }
    __syncthreads();
    cplx akk = A[k + (int64_t)k * m];
    if (cabs1(akk) < tiny) akk = mkc(tiny, 0.0);
    __syncthreads();
    if (tid == 0) A[k + (int64_t)k * m] = akk;
    const cplx inv = cdiv(mkc(1.0, 0.0), akk);
    for (int i = k + 1 + tid; i < m; i += 256) A[i + (int64_t)k * m] = cmul(A[i + (int64_t)k * m], inv);
    __syncthreads();
    const int ti = tid & 63, tj = tid >> 6;
    for (int j = k + 1 + tj; j < m; j += 4) {
      const cplx akj = A[k + (int64_t)j * m];
      for (int i = k + 1 + ti; i < m; i += 64) { cplx a = A[i + (int64_t)j * m]; cfms(a, A[i + (int64_t)k * m], akj); A[i + (int64_t)j * m] = a; }
    }
    __syncthreads();
  }
}

// x <- normalize(A^-1 x) with the stored factors; first != 0: x starts from a seeded random vector.
// Vs [loop][ns][m].
__global__ void __launch_bounds__(256) k_lu_solve(const cplx* __restrict__ LU, const int* __restrict__ piv, int m,
                                                  cplx* __restrict__ Vs, int first) {
  extern __shared__ cplx xs[];   // m
  __shared__ double red[33];
  const int64_t b = blockIdx.x;
  const cplx* A = LU + b * (int64_t)m * m;
  const int* pv = piv + b * (int64_t)m;
  cplx* x = Vs + b * (int64_t)m;
  const int tid = threadIdx.x;
  for (int i = tid; i < m; i += 256)
    xs[i] = first ? mkc(hash_u((uint64_t)b * 0x632BE59BD9B4E019ull + 2 * i), hash_u((uint64_t)b * 0x632BE59BD9B4E019ull + 2 * i + 1)) : x[i];
  __syncthreads();
  if (tid == 0)
    for (int k = 0; k < m; ++k) { const int p = pv[k]; if (p != k) { const cplx t = xs[k]; xs[k] = xs[p]; xs[p] = t; } }
  __syncthreads();
  for (int k = 0; k < m - 1; ++k) {          // L y = P b
    const cplx xk = xs[k];
    for (int i = k + 1 + tid; i < m; i += 256) cfms(xs[i], A[i + (int64_t)k * m], xk);
    __syncthreads();
  }
  for (int k = m - 1; k >= 0; --k) {         // U x = y
    if (tid == 0) xs[k] = cdiv(xs[k], A[k + (int64_t)k * m]);
    __syncthreads();
    const cplx xk = xs[k];
    for (int i = tid; i < k; i += 256) cfms(xs[i], A[i + (int64_t)k * m], xk);
    __syncthreads();
  }
  double ss = 0.0;
  for (int i = tid; i < m; i += 256) ss += cabs2(xs[i]);
  ss = block_sum(ss, red);
  const double sc = ss > 0.0 ? 1.0 / sqrt(ss) : 0.0;
  for (int i = tid; i < m; i += 256) x[i] = cscale(sc, xs[i]);
}

// modified Gram-Schmidt (twice) of the ns vectors of one loop
__global__ void __launch_bounds__(256) k_orth_bands(cplx* __restrict__ Vs, int m, int ns) {
  __shared__ cplx redc[33];
  __shared__ double redd[33];
  cplx* V = Vs + blockIdx.x * (int64_t)ns * m;
  const int tid = threadIdx.x;
  for (int j = 0; j < ns; ++j) {
    cplx* vj = V + (int64_t)j * m;
    for (int pass = 0; pass < 2; ++pass)
      for (int k = 0; k < j; ++k) {
        const cplx* vk = V + (int64_t)k * m;
        cplx d = mkc(0.0, 0.0);
        for (int i = tid; i < m; i += 256) cfmac(d, vk[i], vj[i]);
        d = block_sum(d, redc);
        for (int i = tid; i < m; i += 256) cfms(vj[i], vk[i], d);
        __syncthreads();
      }
    double ss = 0.0;
    for (int i = tid; i < m; i += 256) ss += cabs2(vj[i]);
    ss = block_sum(ss, redd);
    const double sc = ss > 0.0 ? 1.0 / sqrt(ss) : 0.0;
    for (int i = tid; i < m; i += 256) vj[i] = cscale(sc, vj[i]);
    __syncthreads();
  }
}

// phase[b] = arg det A = sum_k arg U_kk + pi * (number of row interchanges), wrapped to (-pi, pi]
__global__ void k_det_phase(const cplx* __restrict__ LU, const int* __restrict__ piv, int m, double* __restrict__ phase) {
  __shared__ double red[33];
  const int64_t b = blockIdx.x;
  const cplx* A = LU + b * (int64_t)m * m;
  const int* pv = piv + b * (int64_t)m;
  double acc = 0.0;
  for (int k = threadIdx.x; k < m; k += blockDim.x) {
    const cplx u = A[k + (int64_t)k * m];
    acc += atan2(u.y, u.x);
    if (pv[k] != k) acc += M_PI;
  }
  acc = block_sum(acc, red);
  if (threadIdx.x == 0) {
    double t = fmod(acc + M_PI, 2.0 * M_PI);
    if (t < 0.0) t += 2.0 * M_PI;
    t -= M_PI;
    if (t <= -M_PI) t = M_PI;
    phase[b] = t;
  }
}

}  // namespace

#define LAUNCH_CHECK() do { ctx->launches++; cudaError_t e__ = cudaGetLastError(); if (e__ != cudaSuccess) return (int)e__; } while (0)

size_t be_nested_general_scratch_bytes(int64_t nl, int m, int ns) {
  return be_align256((size_t)nl * m * m * sizeof(cplx)) + be_align256((size_t)nl * m * sizeof(cplx)) +
         be_align256((size_t)nl * ns * sizeof(cplx)) + be_align256((size_t)nl * ns * m * m * sizeof(cplx)) +
         be_align256((size_t)nl * ns * m * sizeof(int)) + be_align256((size_t)nl * sizeof(int)) + 4096;
}

// W [nl][m][m] column-major (destroyed) -> theta1 [nl][m] sorted on (-pi, pi], Vs [nl][ns][m] orthonormal
// basis of the selected Wannier bands.  Scratch from the context arena.
int be_nested_select_general(be_ctx* ctx, cplx* W, int64_t nl, int m, int wb_lo, int wb_hi, double cut,
                             double* theta1, cplx* Vs) {
  const int ns = wb_hi - wb_lo;
  cudaStream_t st = ctx->stream;
  cplx* Wc = (cplx*)be_arena_alloc(ctx, (size_t)nl * m * m * sizeof(cplx));
  cplx* lam = (cplx*)be_arena_alloc(ctx, (size_t)nl * m * sizeof(cplx));
  cplx* lamS = (cplx*)be_arena_alloc(ctx, (size_t)nl * ns * sizeof(cplx));
  cplx* LU = (cplx*)be_arena_alloc(ctx, (size_t)nl * ns * m * m * sizeof(cplx));
  int* piv = (int*)be_arena_alloc(ctx, (size_t)nl * ns * m * sizeof(int));
  int* fail = (int*)be_arena_alloc(ctx, (size_t)nl * sizeof(int));
  if (!Wc || !lam || !lamS || !LU || !piv || !fail) return BE_ERR_NOMEM;
  BE_CUDA(cudaMemcpyAsync(Wc, W, (size_t)nl * m * m * sizeof(cplx), cudaMemcpyDeviceToDevice, st));
  BE_TRY(be_eigenvalues_general(ctx, W, nl, m, lam, fail));
  BE_TRY(be_sort_phases(ctx, lam, nl, m, theta1, nullptr));
  int nt = ((m + 31) / 32) * 32;
  if (nt > 256) nt = 256;
  k_select_bands<<<(unsigned)nl, nt, (size_t)m * sizeof(double), st>>>(lam, m, wb_lo, ns, cut, lamS);
  LAUNCH_CHECK();
  k_lu_shifted<<<(unsigned)(nl * ns), 256, 0, st>>>(Wc, lamS, m, ns, LU, piv);
  LAUNCH_CHECK();
  const size_t sh = (size_t)m * sizeof(cplx);
  if (sh > 48 * 1024) BE_CUDA(cudaFuncSetAttribute(k_lu_solve, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sh));
  // subspace iteration: every solve is followed by the orthonormalization (degenerate Wannier bands)
  for (int it = 0; it < 3; ++it) {
    k_lu_solve<<<(unsigned)(nl * ns), 256, sh, st>>>(LU, piv, m, Vs, it == 0);
    LAUNCH_CHECK();
    k_orth_bands<<<(unsigned)nl, 256, 0, st>>>(Vs, m, ns);
    LAUNCH_CHECK();
  }
  return BE_OK;
}

// phase [cnt] = arg det of cnt column-major m x m matrices W (not modified), by partially pivoted LU.
int be_det_phase(be_ctx* ctx, const cplx* W, int64_t cnt, int m, double* phase) {
  cplx* LU = (cplx*)be_arena_alloc(ctx, (size_t)cnt * m * m * sizeof(cplx));
  int* piv = (int*)be_arena_alloc(ctx, (size_t)cnt * m * sizeof(int));
  cplx* zero = (cplx*)be_arena_alloc(ctx, (size_t)cnt * sizeof(cplx));
  if (!LU || !piv || !zero) return BE_ERR_NOMEM;
  BE_CUDA(cudaMemsetAsync(zero, 0, (size_t)cnt * sizeof(cplx), ctx->stream));
  k_lu_shifted<<<(unsigned)cnt, 256, 0, ctx->stream>>>(W, zero, m, 1, LU, piv);
  LAUNCH_CHECK();
  k_det_phase<<<(unsigned)cnt, 128, 0, ctx->stream>>>(LU, piv, m, phase);
  LAUNCH_CHECK();
  return BE_OK;
}
