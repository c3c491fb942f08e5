// S1a for matrices that fit shared memory (8 < N <= TS_MAXN): unblocked Householder
// tridiagonalization (zhetd2, lower) with the lower triangle of the matrix resident in one CTA's shared
// memory, packed by columns (35 KB for N = 64, four CTAs per SM with 64 registers per thread; ncu: the
// kernel is bound by shared-memory wavefronts, 67 % of the LSU peak).
// This is the regime of the many-band Wannier-like workload (BASELINE.json configs[4]: 266 240
// matrices of 64 x 64): the lock-step path launches two kernels per column and streams every matrix
// through HBM N times; here a matrix is read once, reduced on chip, and its reflectors are written
// once.  The outputs (d, e, tau, reflectors in the work copy Bw) are exactly those of the blocked
// path, so the tridiagonal eigen-solve and the compact-WY back-transform that follow are shared.
#include "be_common.cuh"

namespace {

constexpr int TS_THREADS = 256;

// packed lower triangle, column by column: element (r, c), r >= c
__device__ __forceinline__ int pk(int r, int c, int N) { return c * N - (c * (c - 1)) / 2 + (r - c); }

// Per column i (n = N - i - 1, x = column i below the diagonal), four barriers:
//   warp 0: zlarfg scalars, reflector v = s x~ to HBM, x~[0] = alpha - beta in place | hemv by all:
//   y = tau s A22 x~ | warp 0: w~ = conj(s) (y - 1/2 tau s^2 (y^H x~) x~) | update by all:
//   A22 -= x~ w~^H + w~ x~^H.  The reflector is not scaled in place: with x~ = x except x~[0] =
//   alpha - beta one has v = s x~, s = 1 / (alpha - beta), so s only multiplies per-row scalars.
// The inner loops walk the packed triangle with running offsets (two integer adds per element).
template <int LGP>
__device__ __forceinline__ void hemv_rows(const cplx* __restrict__ A, const cplx* __restrict__ x, cplx* __restrict__ yb,
                                          cplx ts, int N, int i, int n, int tid) {
  constexpr int P = 1 << LGP;
  const int part = tid & (P - 1);
  constexpr int RPW = 32 >> LGP;                        // rows per warp (an aligned block): warp-uniform trip count
  for (int r = tid >> LGP; r < ((n + RPW - 1) & ~(RPW - 1)); r += TS_THREADS >> LGP) {
    cplx acc = mkc(0.0, 0.0);
    if (r < n) {
      int cc = part;
      int o = pk(i + 1 + r, i + 1 + part, N);           // (r, cc) of the trailing block, cc <= r: along row r
      int step = P * (n - 1 - part) - P * (P - 1) / 2;
      for (; cc <= r; cc += P) { cfma(acc, A[o], x[cc]); o += step; step -= P * P; }
      int o2 = pk(i + 1 + cc, i + 1 + r, N);            // (cc, r), cc > r: down column r, conjugated
      for (; cc < n; cc += P) { cfmac(acc, A[o2], x[cc]); o2 += P; }
    }
#pragma unroll
    for (int m = 1; m < P; m <<= 1) {
      acc.x += __shfl_xor_sync(0xffffffffu, acc.x, m);
      acc.y += __shfl_xor_sync(0xffffffffu, acc.y, m);
    }
    if (part == 0 && r < n) yb[r] = cmul(ts, acc);
  }
}

__global__ void __launch_bounds__(TS_THREADS, 5) k_tridiag_smem(const cplx* __restrict__ H, GridMap map, int64_t loop0,
                                                                cplx* __restrict__ Bw, double* __restrict__ dd,
                                                                double* __restrict__ ee, cplx* __restrict__ tau, int ldn,
                                                                int p0) {
  // The matrix reduced here has order N = ldn - p0: the whole input (p0 = 0, read from H), or the trailing
  // block [p0:, p0:] of the blocked path's work copy Bw (H == nullptr), whose last columns are too short
  // to feed a launch per column.  Outputs go to rows / columns p0 + .. of the ldn-strided arrays.
  const int N = ldn - p0;
  extern __shared__ cplx tsm[];             // A: lower triangle packed by columns (pk), y [N], w~ [N]
  __shared__ cplx sc[3];                    // tau s, -1/2 tau s^2, s
  cplx* A = tsm;
  cplx* yb = tsm + (size_t)N * (N + 1) / 2;
  cplx* wb = yb + N;
  const int64_t c = blockIdx.x;
  const int tid = threadIdx.x, lane = tid & 31;
  cplx* Bc = Bw + c * (int64_t)ldn * ldn + p0 + (int64_t)p0 * ldn;   // element (r, cc) of the block at r + cc * ldn
  if (H) {
    // the row-major Hermitian input read as a column-major array is B = conj(H) (eigh_large.cu)
    const int64_t src = gridmap_index(map, loop0 + c / map.n1, (int)(c % map.n1));
    const cplx* h = H + src * (int64_t)N * N;
    for (int idx = tid; idx < N * N; idx += TS_THREADS) {
      const int r = idx % N, cc = idx / N;
      if (r >= cc) A[pk(r, cc, N)] = h[idx];
    }
  } else {
    for (int idx = tid; idx < N * N; idx += TS_THREADS) {
      const int r = idx % N, cc = idx / N;
      if (r >= cc) A[pk(r, cc, N)] = Bc[r + (int64_t)cc * ldn];
    }
  }
  dd += c * (int64_t)ldn + p0; ee += c * (int64_t)ldn + p0; tau += c * (int64_t)ldn + p0;
  __syncthreads();
  for (int i = 0; i < N - 1; ++i) {
    const int n = N - i - 1;                // order of the trailing block A22 = A[i+1:, i+1:]
    cplx* x = A + pk(i + 1, i, N);          // column i below the diagonal, length n (contiguous)
    if (tid < 32) {
      // ---- zlarfg (warp 0)
      const cplx alpha = x[0];
      double ss = 0.0;
      for (int j = 1 + lane; j < n; j += 32) ss += cabs2(x[j]);
      ss = warp_sum(ss);
      cplx t = mkc(0.0, 0.0), scale = t, amb = t;
      double beta = alpha.x;
      if (ss != 0.0 || alpha.y != 0.0) {
        // in-line reciprocal square root / reciprocals; no rescaling against over/underflow of the
        // squared norm: |H| far from 1e+-150
        const double s2 = cabs2(alpha) + ss;
        const double rs = rsqrt(s2);
        double nrm = s2 * rs;
        nrm = fma(0.5 * rs, fma(-nrm, nrm, s2), nrm);
        beta = -copysign(nrm, alpha.x);
        const double rb = __drcp_rn(beta);
        t = mkc((beta - alpha.x) * rb, -alpha.y * rb);
        amb = mkc(alpha.x - beta, alpha.y);          // real parts of the same sign: no cancellation
        const double q = __drcp_rn(amb.x * amb.x + amb.y * amb.y);
        scale = mkc(amb.x * q, -amb.y * q);
      }
      for (int j = 1 + lane; j < n; j += 32) Bc[(i + 1 + j) + (int64_t)i * ldn] = cmul(scale, x[j]);   // reflector i
      if (lane == 0) {
        const cplx ts = cmul(t, scale);
        sc[0] = ts;
        sc[1] = cmul(mkc(-0.5 * ts.x, -0.5 * ts.y), scale);
        sc[2] = scale;
        dd[i] = A[pk(i, i, N)].x;
        ee[i] = beta;
        tau[i] = t;
        x[0] = amb;
      }
    }
    __syncthreads();
    // ---- y = tau s A22 x~ on the lower triangle: thread = (row, one of P column classes)
    {
      const cplx ts = sc[0];
      if (n > 32) hemv_rows<2>(A, x, yb, ts, N, i, n, tid);
      else if (n > 16) hemv_rows<3>(A, x, yb, ts, N, i, n, tid);
      else if (n > 8) hemv_rows<4>(A, x, yb, ts, N, i, n, tid);
      else hemv_rows<5>(A, x, yb, ts, N, i, n, tid);
    }
    __syncthreads();
    if (tid < 32) {
      // ---- w~ = conj(s) (y - 1/2 tau s^2 (y^H x~) x~)   (warp 0)
      cplx dot = mkc(0.0, 0.0);
      for (int j = lane; j < n; j += 32) cfmac(dot, yb[j], x[j]);
      dot = warp_sum(dot);
      const cplx al = cmul(sc[1], dot), cs = cconj(sc[2]);
      for (int j = lane; j < n; j += 32) { cplx wj = yb[j]; cfma(wj, al, x[j]); wb[j] = cmul(cs, wj); }
    }
    __syncthreads();
    // ---- A22 -= x~ w~^H + w~ x~^H (lower triangle): thread = (row, one of Q column classes)
    {
      const int lgr = n > 32 ? 6 : 5;
      const int q = tid >> lgr, Q = TS_THREADS >> lgr;
      for (int r = tid & ((1 << lgr) - 1); r < n; r += 1 << lgr) {
        const cplx xr = x[r], wr = wb[r];
        int o = pk(i + 1 + r, i + 1 + q, N);
        int step = Q * (n - 1 - q) - Q * (Q - 1) / 2;
        for (int cc = q; cc <= r; cc += Q) {
          cplx a = A[o];
          cfms(a, xr, cconj(wb[cc]));
          cfms(a, wr, cconj(x[cc]));
          A[o] = a;
          o += step; step -= Q * Q;
        }
      }
    }
    __syncthreads();
  }
  if (tid == 0) dd[N - 1] = A[pk(N - 1, N - 1, N)].x;
}


// ---- S1c for the same sizes: X = conj(Q) Z, Q = H_0 H_1 ... H_{N-2}, reflector by reflector with the
// eigenvector columns in REGISTERS.  Eight threads share one column (thread = rows part, part + 8, ...), a
// warp holds four columns; the only communication is the 8-lane butterfly of v^T x, so there is no block
// barrier after the reflectors have been staged (strict lower triangle packed by columns, unit entries
// stored).  Replaces, for N <= TS_MAXN, the compact-WY chain (V extraction, V^H V, T, three GEMMs), whose
// 64 x 64 operands made it HBM bound at ~1 MB of traffic per matrix.
//   The work matrix is B = conj(H) (see above), so eigenvectors of H are conj(Q) Z:
//   x[i+1:] -= conj(tau_i) conj(v_i) (v_i^T x[i+1:]),  i = N-2 .. 0,  x real on entry.
template <int RPT>
__global__ void __launch_bounds__(256, RPT <= 8 ? 3 : 2) k_backtransform_small(const cplx* __restrict__ Bw, const cplx* __restrict__ tau,
                                                                const double* __restrict__ Z, cplx* __restrict__ X,
                                                                int N, int nv) {
  extern __shared__ cplx bsm[];             // V packed: column i holds rows i+1 .. N-1 at i (N-1) - i (i-1)/2
  cplx* vs = bsm;
  cplx* tc = bsm + (size_t)N * (N - 1) / 2;   // conj(tau) [N]
  const int64_t c = blockIdx.x;
  const int tid = threadIdx.x, part = tid & 7;
  const int j = blockIdx.y * 32 + (tid >> 3);
  const cplx* Bc = Bw + c * (int64_t)N * N;
  for (int idx = tid; idx < N * N; idx += 256) {
    const int r = idx % N, i = idx / N;
    if (r > i && i < N - 1) vs[i * (N - 1) - (i * (i - 1)) / 2 + (r - i - 1)] = (r == i + 1) ? mkc(1.0, 0.0) : Bc[idx];
  }
  for (int i = tid; i < N - 1; i += 256) tc[i] = cconj(tau[c * N + i]);
  cplx z[RPT];
#pragma unroll
  for (int k = 0; k < RPT; ++k) {
    const int r = part + 8 * k;
    z[k] = (r < N && j < nv) ? mkc(Z[c * (int64_t)N * nv + (int64_t)r * nv + j], 0.0) : mkc(0.0, 0.0);
  }
  __syncthreads();
  for (int i = N - 2; i >= 0; --i) {
    const cplx* v = vs + i * (N - 1) - (i * (i - 1)) / 2 - (i + 1);   // v[r], r = i+1 .. N-1
    cplx d0 = mkc(0.0, 0.0), d1 = mkc(0.0, 0.0);
#pragma unroll
    for (int k = 0; k < RPT; ++k) {
      if (8 * k + 7 > i) {
        const int r = part + 8 * k;
        if (r > i && r < N) { if (k & 1) cfma(d1, v[r], z[k]); else cfma(d0, v[r], z[k]); }
      }
    }
    d0 = cadd(d0, d1);
#pragma unroll
    for (int m = 1; m < 8; m <<= 1) {
      d0.x += __shfl_xor_sync(0xffffffffu, d0.x, m);
      d0.y += __shfl_xor_sync(0xffffffffu, d0.y, m);
    }
    const cplx g = cmul(tc[i], d0);
#pragma unroll
    for (int k = 0; k < RPT; ++k) {
      if (8 * k + 7 > i) {
        const int r = part + 8 * k;
        if (r > i && r < N) cfms(z[k], cconj(v[r]), g);
      }
    }
  }
  if (j < nv) {
    cplx* Xc = X + c * (int64_t)N * nv + (int64_t)j * N;
#pragma unroll
    for (int k = 0; k < RPT; ++k) {
      const int r = part + 8 * k;
      if (r < N) Xc[r] = z[k];
    }
  }
}

}  // namespace

int be_tridiag_small(be_ctx* ctx, const cplx* H, const GridMap& map, int64_t loop0, int64_t cnt, int N, cplx* Bw,
                     double* d, double* e, cplx* tau, int p0) {
  const int ns = N - p0;   // order of the matrix reduced on chip (H == nullptr: trailing block of Bw)
  if (ns > TS_MAXN || ns < 1 || (H && p0 != 0)) return BE_ERR_UNSUPPORTED;
  const size_t sh = ((size_t)ns * (ns + 1) / 2 + 2 * ns) * sizeof(cplx);
  if (sh > 48 * 1024) BE_CUDA(cudaFuncSetAttribute(k_tridiag_smem, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sh));
  // six CTAs of 35 KB per SM need the full shared-memory carve-out
  BE_CUDA(cudaFuncSetAttribute(k_tridiag_smem, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
  be_prof_begin(ctx, PK_HEMV);
  k_tridiag_smem<<<(unsigned)cnt, TS_THREADS, sh, ctx->stream>>>(H, map, loop0, Bw, d, e, tau, N, p0);
  be_prof_end(ctx, PK_HEMV, (double)cnt * ns * ns * 32.0, (double)cnt * (16.0 / 3.0) * ns * (double)ns * ns);
  ctx->launches++;
  return (int)cudaGetLastError();
}

int be_backtransform_small(be_ctx* ctx, const cplx* Bw, const cplx* tau, const double* Z, cplx* X, int64_t cnt, int N,
                           int nv) {
  if (N > TS_MAXN) return BE_ERR_UNSUPPORTED;
  const size_t sh = ((size_t)N * (N - 1) / 2 + N) * sizeof(cplx);
  const dim3 grid((unsigned)cnt, (unsigned)((nv + 31) / 32));
  be_prof_begin(ctx, PK_GEMM);
  if (N <= 64) {
    if (sh > 48 * 1024) BE_CUDA(cudaFuncSetAttribute(k_backtransform_small<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sh));
    BE_CUDA(cudaFuncSetAttribute(k_backtransform_small<8>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
    k_backtransform_small<8><<<grid, 256, sh, ctx->stream>>>(Bw, tau, Z, X, N, nv);
  } else {
    BE_CUDA(cudaFuncSetAttribute(k_backtransform_small<13>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sh));
    k_backtransform_small<13><<<grid, 256, sh, ctx->stream>>>(Bw, tau, Z, X, N, nv);
  }
  be_prof_end(ctx, PK_GEMM, (double)cnt * (16.0 * N * N + 24.0 * N * nv), (double)cnt * 8.0 * N * (double)N * nv);
  ctx->launches++;
  return (int)cudaGetLastError();
}
