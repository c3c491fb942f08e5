// S1a for matrices that fit shared memory (8 < N <= TS_MAXN): unblocked Householder
// tridiagonalization (zhetd2, lower) with the whole matrix resident in one CTA's shared memory.
// This is the regime of the many-band Wannier-like workload (BASELINE.json configs[4]: 266 240
// matrices of 64 x 64): the lock-step path launches two kernels per column and streams every matrix
// through HBM N times; here a matrix is read once, reduced on chip, and its reflectors are written
// once.  The outputs (d, e, tau, reflectors in the work copy Bw) are exactly those of the blocked
// path, so the tridiagonal eigen-solve and the compact-WY back-transform that follow are shared.
#include "be_common.cuh"

namespace {

constexpr int TS_THREADS = 256;

// Block-wide sum with ONE barrier: per-warp partials go to one of two alternating buffers (the next use
// of the same buffer is two reductions, hence at least one barrier, later), every thread adds the 8 partials.
__device__ __forceinline__ double block_sum1(double v, double* buf, int& par) {
  v = warp_sum(v);
  if ((threadIdx.x & 31) == 0) buf[par * 8 + (threadIdx.x >> 5)] = v;
  __syncthreads();
  double t = buf[par * 8];
#pragma unroll
  for (int w = 1; w < TS_THREADS / 32; ++w) t += buf[par * 8 + w];
  par ^= 1;
  return t;
}
__device__ __forceinline__ cplx block_sum1(cplx v, cplx* buf, int& par) {
  v = warp_sum(v);
  if ((threadIdx.x & 31) == 0) buf[par * 8 + (threadIdx.x >> 5)] = v;
  __syncthreads();
  cplx t = buf[par * 8];
#pragma unroll
  for (int w = 1; w < TS_THREADS / 32; ++w) t = cadd(t, buf[par * 8 + w]);
  par ^= 1;
  return t;
}

__global__ void __launch_bounds__(TS_THREADS) k_tridiag_smem(const cplx* __restrict__ H, GridMap map, int64_t loop0,
                                                             cplx* __restrict__ Bw, double* __restrict__ dd,
                                                             double* __restrict__ ee, cplx* __restrict__ tau, int N) {
  extern __shared__ cplx tsm[];             // A [N][ld] column-major (ld = N + 1: conflict-free column walks), w [N]
  __shared__ double redd[16];
  __shared__ cplx redc[16];
  int pard = 0, parc = 0;
  const int ld = N + 1;
  cplx* A = tsm;
  cplx* w = tsm + (size_t)N * ld;
  const int64_t c = blockIdx.x;
  const int tid = threadIdx.x;
  {
    // the row-major Hermitian input read as a column-major array is B = conj(H) (eigh_large.cu)
    const int64_t src = gridmap_index(map, loop0 + c / map.n1, (int)(c % map.n1));
    const cplx* h = H + src * (int64_t)N * N;
    for (int idx = tid; idx < N * N; idx += TS_THREADS) {
      const int r = idx % N, cc = idx / N;
      A[r + cc * ld] = h[idx];
    }
  }
  __syncthreads();
  for (int i = 0; i < N - 1; ++i) {
    const int n = N - i - 1;                // order of the trailing block A22 = A[i+1:, i+1:]
    cplx* x = A + (i + 1) + i * ld;         // column i below the diagonal, length n
    // ---- zlarfg
    double ss = 0.0;
    for (int r = 1 + tid; r < n; r += TS_THREADS) ss += cabs2(x[r]);
    const cplx alpha = x[0];                 // not modified before the next barrier
    const double xn2 = block_sum1(ss, redd, pard);
    double beta; cplx t;
    if (xn2 == 0.0 && alpha.y == 0.0) {
      beta = alpha.x; t = mkc(0.0, 0.0);
    } else {
      beta = -copysign(sqrt(cabs2(alpha) + xn2), alpha.x);
      t = mkc((beta - alpha.x) / beta, -alpha.y / beta);
      const cplx scale = cdiv(mkc(1.0, 0.0), mkc(alpha.x - beta, alpha.y));
      for (int r = 1 + tid; r < n; r += TS_THREADS) x[r] = cmul(x[r], scale);
    }
    if (tid == 0) {
      x[0] = mkc(1.0, 0.0);
      dd[c * N + i] = A[i + i * ld].x;
      ee[c * N + i] = beta;
      tau[c * N + i] = t;
    }
    __syncthreads();
    if (t.x == 0.0 && t.y == 0.0) continue;   // H_i = 1 (uniform over the CTA)
    // ---- y = tau A22 v on the lower triangle: thread = (row, quarter of the columns)
    const cplx* A22 = A + (i + 1) + (i + 1) * ld;
    for (int r0 = 0; r0 < n; r0 += TS_THREADS / 4) {
      const int r = r0 + (tid >> 2), part = tid & 3;
      cplx acc = mkc(0.0, 0.0);
      if (r < n)
        for (int cc = part; cc < n; cc += 4) {
          if (cc <= r) cfma(acc, A22[r + cc * ld], x[cc]);
          else cfmac(acc, A22[cc + r * ld], x[cc]);
        }
      acc.x += __shfl_xor_sync(0xffffffffu, acc.x, 1); acc.y += __shfl_xor_sync(0xffffffffu, acc.y, 1);
      acc.x += __shfl_xor_sync(0xffffffffu, acc.x, 2); acc.y += __shfl_xor_sync(0xffffffffu, acc.y, 2);
      if (r < n && part == 0) w[r] = cmul(t, acc);
    }
    __syncthreads();
    // ---- w += -1/2 tau (w^H v) v
    cplx dot = mkc(0.0, 0.0);
    for (int r = tid; r < n; r += TS_THREADS) cfmac(dot, w[r], x[r]);
    dot = block_sum1(dot, redc, parc);
    const cplx al = cmul(mkc(-0.5 * t.x, -0.5 * t.y), dot);
    for (int r = tid; r < n; r += TS_THREADS) { cplx wr = w[r]; cfma(wr, al, x[r]); w[r] = wr; }
    __syncthreads();
    // ---- A22 -= v w^H + w v^H (lower triangle): thread = (row, quarter of the columns)
    cplx* A22w = A + (i + 1) + (i + 1) * ld;
    for (int r0 = 0; r0 < n; r0 += 64) {
      const int r = r0 + (tid & 63);
      if (r < n) {
        const cplx vr = x[r], wr = w[r];
        for (int cc = tid >> 6; cc <= r; cc += 4) {
          cplx a = A22w[r + cc * ld];
          cfms(a, vr, cconj(w[cc]));
          cfms(a, wr, cconj(x[cc]));
          A22w[r + cc * ld] = a;
        }
      }
    }
    __syncthreads();
  }
  if (tid == 0) dd[c * N + N - 1] = A[(N - 1) + (N - 1) * ld].x;
  // reflectors (and the rest of the work copy) for the back-transform
  cplx* Bc = Bw + c * (int64_t)N * N;
  for (int idx = tid; idx < N * N; idx += TS_THREADS) {
    const int r = idx % N, cc = idx / N;
    Bc[idx] = A[r + cc * ld];
  }
}

}  // namespace

int be_tridiag_small(be_ctx* ctx, const cplx* H, const GridMap& map, int64_t loop0, int64_t cnt, int N, cplx* Bw,
                     double* d, double* e, cplx* tau) {
  if (N > TS_MAXN) return BE_ERR_UNSUPPORTED;
  const size_t sh = ((size_t)N * (N + 1) + N) * sizeof(cplx);
  if (sh > 48 * 1024) BE_CUDA(cudaFuncSetAttribute(k_tridiag_smem, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sh));
  be_prof_begin(ctx, PK_HEMV);
  k_tridiag_smem<<<(unsigned)cnt, TS_THREADS, sh, ctx->stream>>>(H, map, loop0, Bw, d, e, tau, N);
  be_prof_end(ctx, PK_HEMV, (double)cnt * N * N * 32.0, (double)cnt * (16.0 / 3.0) * N * (double)N * N);
  ctx->launches++;
  return (int)cudaGetLastError();
}
