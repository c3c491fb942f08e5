// S1b -- orthogonalization of the inverse-iteration vectors inside clusters of close eigenvalues.
//
// Vectors of eigenvalues a gap g apart come out of inverse iteration orthogonal to ~eps ||T|| / g;
// inside a cluster (gap <= ctol ||T||, same unreduced block of T) they have to be orthogonalized
// explicitly.  Two regimes, all matrices of the chunk in one launch each:
//   * small clusters (< BIGC vectors; the generic case, a few dozen per matrix): classical
//     Gram-Schmidt applied twice, one CTA per matrix walking its list of small clusters;
//   * big clusters (exactly degenerate spectra: the projected spin operator P S P has eigenvalues
//     +-1 with multiplicity n_occ / 2 when [H, S] = 0): Cholesky-QR on the FP64
//     tensor cores -- G = Z_c^T Z_c (grouped real DMMA GEMM over all big clusters of all matrices),
//     G = R^T R and R^-1 per cluster, Z_c <- Z_c R^-1 (second grouped GEMM).  Sequential Gram-Schmidt
//     on a 400-vector cluster costs 125 ms per matrix; this costs N L^2 flops at GEMM rate.
// Z is [N][nv] row-major per matrix (vector index fastest), real.
#include "be_common.cuh"
#include <float.h>

namespace {

constexpr int BIGC = 16;    // clusters of at least BIGC vectors take the Cholesky-QR path
constexpr int GT = 64;      // tile of the grouped GEMMs
constexpr int GK = 16;
constexpr int GLD = 68;     // [k][mn] layout, GLD % 16 == 4
constexpr int GLDK = 20;    // [mn][k] layout

__device__ __forceinline__ void dmma_r(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

// Per-matrix cluster lists.
struct ClusterBufs {
  int* perm;      // [cnt][nv]   vectors ordered by (block, eigenvalue index)
  int* nsmall;    // [cnt]
  int2* small;    // [cnt][nv/2 + 1]     {start in perm, length}
  int* nbig;      // [cnt]
  int4* big;      // [cnt][maxbig]       {start in perm, length, r0, r1}
  int* goff;      // [cnt][maxbig]       offset (doubles) of the cluster's L x L matrix in G
  double* G;      // [cnt][nv * nv]
  double* Zt;     // [cnt][N * nv]
};

// ------------------------------------------------------------------------------------------
// perm, then the cluster scan (sequential over the nv eigenvalues of one matrix).
__global__ void __launch_bounds__(256) k_find_clusters(const double* __restrict__ lam, const double* __restrict__ tnorm,
                                                       const int* __restrict__ blk, int N, int nv, double ctol,
                                                       int maxbig, ClusterBufs cb) {
  const int64_t c = blockIdx.x;
  const int* bk = blk + c * (int64_t)nv * 2;
  int* perm = cb.perm + c * (int64_t)nv;
  const double* l = lam + c * N;
  const int tid = threadIdx.x;
  // order by (block, eigenvalue index): close eigenvalues of one unreduced block become neighbours
  // even when eigenvalues of other blocks lie between them
  for (int v = tid; v < nv; v += 256) {
    const int b = bk[2 * v];
    int rank = 0;
    for (int u = 0; u < nv; ++u) { const int bu = bk[2 * u]; rank += (bu < b) || (bu == b && u < v); }
    perm[rank] = v;
  }
  __syncthreads();
  if (tid != 0) return;
  const double gaptol = ctol * tnorm[c];
  int2* sm = cb.small + c * (int64_t)(nv / 2 + 1);
  int4* bg = cb.big + c * (int64_t)maxbig;
  int* go = cb.goff + c * (int64_t)maxbig;
  int ns = 0, nb = 0, off = 0, s = 0;
  while (s < nv) {
    int e = s + 1;
    const int bs = bk[2 * perm[s]];
    while (e < nv && bk[2 * perm[e]] == bs && l[perm[e]] - l[perm[e - 1]] <= gaptol) ++e;
    const int len = e - s;
    if (len >= BIGC && nb < maxbig) {
      bg[nb] = make_int4(s, len, bs, bk[2 * perm[s] + 1] + 1);
      go[nb] = off;
      off += len * len;
      ++nb;
    } else if (len > 1) {
      sm[ns++] = make_int2(s, len);
    }
    s = e;
  }
  cb.nsmall[c] = ns;
  cb.nbig[c] = nb;
}

// ------------------------------------------------------------------------------------------
// Small clusters: classical Gram-Schmidt applied twice; gridDim.y CTAs per matrix share its clusters round robin
// (the clusters own disjoint columns; one CTA per matrix walked them one after the other: 6.4 ms per launch on the
// bench workload).
constexpr int ORTH_SMALL_SPLIT = 4;
__global__ void __launch_bounds__(256) k_orth_small(const int* __restrict__ blk, double* __restrict__ Z, int N, int nv,
                                                    ClusterBufs cb, int* __restrict__ info) {
  __shared__ double red[33];
  __shared__ double coef[BIGC];
  __shared__ int cols[BIGC];
  const int64_t c = blockIdx.x;
  const int* bk = blk + c * (int64_t)nv * 2;
  const int* perm = cb.perm + c * (int64_t)nv;
  const int2* sm = cb.small + c * (int64_t)(nv / 2 + 1);
  const int ns = cb.nsmall[c];
  const int tid = threadIdx.x;
  double* Zc = Z + c * (int64_t)N * nv;
  for (int q = blockIdx.y; q < ns; q += gridDim.y) {
    const int s0 = sm[q].x, len = sm[q].y;
    const int r0 = bk[2 * perm[s0]], r1 = bk[2 * perm[s0] + 1] + 1;   // support of the cluster's block
    if (len > BIGC) {
      // overflow of the big-cluster list (never with the default sizes): generic slow path
      for (int j = 0; j < len; ++j) {
        const int cj = perm[s0 + j];
        for (int pass = 0; pass < 2 && j > 0; ++pass)
          for (int k = 0; k < j; ++k) {
            const int ck = perm[s0 + k];
            double acc = 0.0;
            for (int r = r0 + tid; r < r1; r += 256) acc = fma(Zc[(int64_t)r * nv + ck], Zc[(int64_t)r * nv + cj], acc);
            acc = block_sum(acc, red);
            for (int r = r0 + tid; r < r1; r += 256) Zc[(int64_t)r * nv + cj] -= acc * Zc[(int64_t)r * nv + ck];
            __syncthreads();
          }
        double ss = 0.0;
        for (int r = r0 + tid; r < r1; r += 256) { const double z = Zc[(int64_t)r * nv + cj]; ss = fma(z, z, ss); }
        ss = block_sum(ss, red);
        const double sc = (ss > 0.0) ? 1.0 / sqrt(ss) : 0.0;
        for (int r = r0 + tid; r < r1; r += 256) Zc[(int64_t)r * nv + cj] *= sc;
        __syncthreads();
      }
      continue;
    }
    if (tid < len) cols[tid] = perm[s0 + tid];
    __syncthreads();
    for (int j = 0; j < len; ++j) {
      const int cj = cols[j];
      for (int pass = 0; pass < 2 && j > 0; ++pass) {
        // r_k = sum_i Z[i][col k] Z[i][col j], k < j  (j < BIGC = 16 accumulators)
        double acc[BIGC];
#pragma unroll
        for (int k = 0; k < BIGC; ++k) acc[k] = 0.0;
        for (int r = r0 + tid; r < r1; r += 256) {
          const double zj = Zc[(int64_t)r * nv + cj];
#pragma unroll
          for (int k = 0; k < BIGC; ++k)
            if (k < j) acc[k] = fma(Zc[(int64_t)r * nv + cols[k]], zj, acc[k]);
        }
#pragma unroll
        for (int k = 0; k < BIGC; ++k)
          if (k < j) {
            const double t = block_sum(acc[k], red);
            if (tid == 0) coef[k] = t;
          }
        __syncthreads();
        for (int r = r0 + tid; r < r1; r += 256) {
          double zj = Zc[(int64_t)r * nv + cj];
          for (int k = 0; k < j; ++k) zj = fma(-coef[k], Zc[(int64_t)r * nv + cols[k]], zj);
          Zc[(int64_t)r * nv + cj] = zj;
        }
        __syncthreads();
      }
      double ss = 0.0;
      for (int r = r0 + tid; r < r1; r += 256) { const double z = Zc[(int64_t)r * nv + cj]; ss = fma(z, z, ss); }
      ss = block_sum(ss, red);
      if (j > 0 && ss < 1e-20 && tid == 0 && info) atomicAdd(&info[c], 1);   // dependent start vectors
      const double sc = (ss > 0.0) ? 1.0 / sqrt(ss) : 0.0;
      for (int r = r0 + tid; r < r1; r += 256) Zc[(int64_t)r * nv + cj] *= sc;
      __syncthreads();
    }
  }
}

// ------------------------------------------------------------------------------------------
// Grouped real GEMMs on DMMA.  CTA = 256 threads = 8 warps as 2 (M) x 4 (N), CTA tile 64 x 64,
// warp tile 32 x 16 = 4 x 2 blocks of m8n8k4; operands staged through shared memory.

// locate work item t of matrix c: big cluster q and local tile index; returns false if t is past the end
__device__ __forceinline__ bool find_cluster(const ClusterBufs& cb, int64_t c, int maxbig, int t, bool gram, int N,
                                             int& q, int& tl) {
  const int nb = cb.nbig[c];
  const int4* bg = cb.big + c * (int64_t)maxbig;
  for (q = 0; q < nb; ++q) {
    const int L = bg[q].y, tq = (L + GT - 1) / GT;
    const int rows = bg[q].w - bg[q].z;
    const int nt = gram ? tq * (tq + 1) / 2 : tq * ((rows + GT - 1) / GT);
    if (t < nt) { tl = t; return true; }
    t -= nt;
  }
  (void)N;
  return false;
}

__device__ __forceinline__ void mma_tile(const double* As, const double* Bs, bool b_kcontig, int warp, int lane,
                                         double (&acc)[4][2][2]) {
  const int wm = warp & 1, wn = warp >> 1, g = lane >> 2, tg = lane & 3;
#pragma unroll
  for (int ks = 0; ks < GK / 4; ++ks) {
    const int k = ks * 4 + tg;
    double a[4], b[2];
#pragma unroll
    for (int mb = 0; mb < 4; ++mb) a[mb] = As[k * GLD + wm * 32 + mb * 8 + g];
#pragma unroll
    for (int nb = 0; nb < 2; ++nb) {
      const int n = wn * 16 + nb * 8 + g;
      b[nb] = b_kcontig ? Bs[n * GLDK + k] : Bs[k * GLD + n];
    }
#pragma unroll
    for (int mb = 0; mb < 4; ++mb)
#pragma unroll
      for (int nb = 0; nb < 2; ++nb) dmma_r(acc[mb][nb][0], acc[mb][nb][1], a[mb], b[nb]);
  }
}

// G_q[i][j] = sum_r Z[r][col_i] Z[r][col_j], r in the block's support; tiles on or below the
// diagonal are computed and mirrored.
__global__ void __launch_bounds__(256) k_cgram(const double* __restrict__ Z, int N, int nv, int maxbig, int tmaxg,
                                               ClusterBufs cb) {
  __shared__ double As[GK * GLD], Bs[GK * GLD];
  __shared__ int colA[GT], colB[GT];
  const int64_t c = blockIdx.x / tmaxg;
  int q, tl;
  if (!find_cluster(cb, c, maxbig, blockIdx.x % tmaxg, true, N, q, tl)) return;
  const int4 d = cb.big[c * (int64_t)maxbig + q];
  const int s0 = d.x, L = d.y, r0 = d.z, r1 = d.w;
  int ti = 0;
  while ((ti + 1) * (ti + 2) / 2 <= tl) ++ti;
  const int tj = tl - ti * (ti + 1) / 2;
  const int* perm = cb.perm + c * (int64_t)nv;
  const double* Zc = Z + c * (int64_t)N * nv;
  double* G = cb.G + c * (int64_t)nv * nv + cb.goff[c * (int64_t)maxbig + q];
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  if (tid < GT) {
    const int i = ti * GT + tid, j = tj * GT + tid;
    colA[tid] = (i < L) ? perm[s0 + i] : -1;
    colB[tid] = (j < L) ? perm[s0 + j] : -1;
  }
  __syncthreads();
  double acc[4][2][2];
#pragma unroll
  for (int a = 0; a < 4; ++a)
#pragma unroll
    for (int b = 0; b < 2; ++b) acc[a][b][0] = acc[a][b][1] = 0.0;
  const int li = tid & 63, lk = tid >> 6;
  const int ca = colA[li], cbj = colB[li];
  for (int k0 = r0; k0 < r1; k0 += GK) {
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int k = lk + 4 * u, r = k0 + k;
      const bool ok = r < r1;
      As[k * GLD + li] = (ok && ca >= 0) ? Zc[(int64_t)r * nv + ca] : 0.0;
      Bs[k * GLD + li] = (ok && cbj >= 0) ? Zc[(int64_t)r * nv + cbj] : 0.0;
    }
    __syncthreads();
    mma_tile(As, Bs, false, warp, lane, acc);
    __syncthreads();
  }
  const int wm = warp & 1, wn = warp >> 1, g = lane >> 2, tg = lane & 3;
#pragma unroll
  for (int mb = 0; mb < 4; ++mb)
#pragma unroll
    for (int nb = 0; nb < 2; ++nb)
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const int i = ti * GT + wm * 32 + mb * 8 + g, j = tj * GT + wn * 16 + nb * 8 + 2 * tg + e;
        if (i < L && j < L) {
          G[(int64_t)i * L + j] = acc[mb][nb][e];
          if (ti != tj) G[(int64_t)j * L + i] = acc[mb][nb][e];
        }
      }
}

// ------------------------------------------------------------------------------------------
// Per big cluster: G = R^T R (Cholesky-Crout, row by row, in place in the upper triangle), then
// X = R^-1 in place (column by column).  One CTA per cluster; G stays in L2.
constexpr int CHT = 512;   // threads of k_chol_inv
__global__ void __launch_bounds__(CHT) k_chol_inv(int nv, int maxbig, ClusterBufs cb, int* __restrict__ info) {
  extern __shared__ double colk[];   // L doubles
  __shared__ int s_fail;
  const int64_t c = blockIdx.x / maxbig;
  const int q = blockIdx.x % maxbig;
  if (q >= cb.nbig[c]) return;
  const int L = cb.big[c * (int64_t)maxbig + q].y;
  double* G = cb.G + c * (int64_t)nv * nv + cb.goff[c * (int64_t)maxbig + q];
  const int tid = threadIdx.x;
  if (tid == 0) s_fail = 0;
  for (int k = 0; k < L; ++k) {
    for (int p = tid; p < k; p += CHT) colk[p] = G[(int64_t)p * L + k];   // R[0:k, k]
    __syncthreads();
    for (int j = k + tid; j < L; j += CHT) {
      double t0 = G[(int64_t)k * L + j], t1 = 0.0;
      int p = 0;
      for (; p + 1 < k; p += 2) {
        t0 = fma(-colk[p], G[(int64_t)p * L + j], t0);
        t1 = fma(-colk[p + 1], G[(int64_t)(p + 1) * L + j], t1);
      }
      if (p < k) t0 = fma(-colk[p], G[(int64_t)p * L + j], t0);
      G[(int64_t)k * L + j] = t0 + t1;
    }
    __syncthreads();
    double d = G[(int64_t)k * L + k];
    if (!(d > 1e-13)) { d = 1.0; if (tid == 0) s_fail = 1; }   // vectors are normalized: G[k][k] started at 1
    const double rs = 1.0 / sqrt(d);
    __syncthreads();
    for (int j = k + tid; j < L; j += CHT) {
      const double t = G[(int64_t)k * L + j];
      G[(int64_t)k * L + j] = (j == k) ? d * rs : t * rs;
    }
    __syncthreads();
  }
  if (s_fail) {   // numerically dependent vectors: leave the cluster as it is (identity), flag the matrix
    for (int idx = tid; idx < L * L; idx += CHT) G[idx] = (idx / L == idx % L) ? 1.0 : 0.0;
    if (tid == 0 && info) atomicAdd(&info[c], 1);
    return;
  }
  // X = R^-1, upper triangular, column j: X[j][j] = 1 / R[j][j], X[i][j] = -(sum_{k=i}^{j-1} X[i][k] R[k][j]) X[j][j]
  for (int j = 0; j < L; ++j) {
    for (int k = tid; k < j; k += CHT) colk[k] = G[(int64_t)k * L + j];
    __syncthreads();
    const double xjj = 1.0 / G[(int64_t)j * L + j];
    __syncthreads();
    for (int i = tid; i <= j; i += CHT) {
      if (i == j) { G[(int64_t)j * L + j] = xjj; continue; }
      double t0 = 0.0, t1 = 0.0;
      const double* xi = G + (int64_t)i * L;
      int k = i;
      for (; k + 1 < j; k += 2) { t0 = fma(xi[k], colk[k], t0); t1 = fma(xi[k + 1], colk[k + 1], t1); }
      if (k < j) t0 = fma(xi[k], colk[k], t0);
      G[(int64_t)i * L + j] = -(t0 + t1) * xjj;
    }
    __syncthreads();
  }
}

// Zt[r][col_i] = sum_{j <= i} X[j][i] Z[r][col_j]   (Z_c <- Z_c R^-1), tile = 64 vectors x 64 rows.
__global__ void __launch_bounds__(256) k_cupdate(const double* __restrict__ Z, int N, int nv, int maxbig, int tmaxu,
                                                 ClusterBufs cb) {
  __shared__ double As[GK * GLD], Bs[GT * GLDK];
  const int64_t c = blockIdx.x / tmaxu;
  int q, tl;
  if (!find_cluster(cb, c, maxbig, blockIdx.x % tmaxu, false, N, q, tl)) return;
  const int4 d = cb.big[c * (int64_t)maxbig + q];
  const int s0 = d.x, L = d.y, r0 = d.z, r1 = d.w;
  const int tq = (L + GT - 1) / GT;
  const int ti = tl % tq, tr = tl / tq;
  const int* perm = cb.perm + c * (int64_t)nv + s0;
  const double* Zc = Z + c * (int64_t)N * nv;
  double* Zt = cb.Zt + c * (int64_t)N * nv;
  const double* X = cb.G + c * (int64_t)nv * nv + cb.goff[c * (int64_t)maxbig + q];
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  double acc[4][2][2];
#pragma unroll
  for (int a = 0; a < 4; ++a)
#pragma unroll
    for (int b = 0; b < 2; ++b) acc[a][b][0] = acc[a][b][1] = 0.0;
  const int li = tid & 63, lk = tid >> 6;          // A staging: (vector i, k)
  const int bk = tid & 15, bn = tid >> 4;          // B staging: (k, row n)
  const int i = ti * GT + li;
  const int kend = ((ti + 1) * GT < L) ? (ti + 1) * GT : L;   // X is upper triangular: j <= i
  for (int k0 = 0; k0 < kend; k0 += GK) {
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int j = k0 + lk + 4 * u;
      As[(lk + 4 * u) * GLD + li] = (j < L && i < L && j <= i) ? X[(int64_t)j * L + i] : 0.0;
    }
    {
      const int j = k0 + bk;
      const int col = (j < L) ? perm[j] : -1;
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int n = bn + 16 * u, r = r0 + tr * GT + n;
        Bs[n * GLDK + bk] = (col >= 0 && r < r1) ? Zc[(int64_t)r * nv + col] : 0.0;
      }
    }
    __syncthreads();
    mma_tile(As, Bs, true, warp, lane, acc);
    __syncthreads();
  }
  const int wm = warp & 1, wn = warp >> 1, g = lane >> 2, tg = lane & 3;
#pragma unroll
  for (int mb = 0; mb < 4; ++mb) {
    const int io = ti * GT + wm * 32 + mb * 8 + g;
    if (io >= L) continue;
    const int col = perm[io];
#pragma unroll
    for (int nb = 0; nb < 2; ++nb)
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const int r = r0 + tr * GT + wn * 16 + nb * 8 + 2 * tg + e;
        if (r < r1) Zt[(int64_t)r * nv + col] = acc[mb][nb][e];
      }
  }
}

__global__ void __launch_bounds__(256) k_ccopy(double* __restrict__ Z, int N, int nv, int maxbig, ClusterBufs cb) {
  const int64_t c = blockIdx.x / maxbig;
  const int q = blockIdx.x % maxbig;
  if (q >= cb.nbig[c]) return;
  const int4 d = cb.big[c * (int64_t)maxbig + q];
  const int s0 = d.x, L = d.y, r0 = d.z, r1 = d.w;
  const int* perm = cb.perm + c * (int64_t)nv + s0;
  double* Zc = Z + c * (int64_t)N * nv;
  const double* Zt = cb.Zt + c * (int64_t)N * nv;
  const int64_t tot = (int64_t)(r1 - r0) * L;
  for (int64_t idx = threadIdx.x; idx < tot; idx += 256) {
    const int r = r0 + (int)(idx / L), col = perm[idx % L];
    Zc[(int64_t)r * nv + col] = Zt[(int64_t)r * nv + col];
  }
}

}  // namespace

// ------------------------------------------------------------------------------------------
static int maxbig_of(int nv) { return nv / BIGC + 1; }

static size_t cluster_carve(char* base, int64_t cnt, int N, int nv, ClusterBufs* cb) {
  size_t off = 0;
  auto take = [&](size_t bytes) { char* p = base ? base + off : nullptr; off += be_align256(bytes); return p; };
  const int mb = maxbig_of(nv);
  ClusterBufs b;
  b.perm = (int*)take(cnt * (size_t)nv * sizeof(int));
  b.nsmall = (int*)take(cnt * sizeof(int));
  b.small = (int2*)take(cnt * (size_t)(nv / 2 + 1) * sizeof(int2));
  b.nbig = (int*)take(cnt * sizeof(int));
  b.big = (int4*)take(cnt * (size_t)mb * sizeof(int4));
  b.goff = (int*)take(cnt * (size_t)mb * sizeof(int));
  b.G = (double*)take(cnt * (size_t)nv * nv * sizeof(double));
  b.Zt = (double*)take(cnt * (size_t)N * nv * sizeof(double));
  if (cb) *cb = b;
  return off;
}

size_t be_cluster_orth_scratch_bytes(int64_t cnt, int N, int nv) {
  return nv > 0 ? cluster_carve(nullptr, cnt, N, nv, nullptr) : 0;
}

#define LAUNCH_CHECK() do { ctx->launches++; cudaError_t e__ = cudaGetLastError(); if (e__ != cudaSuccess) return (int)e__; } while (0)

// lam [cnt][N] eigenvalues, tnorm [cnt], blk [cnt][nv][2] block of each vector, Z [cnt][N][nv].
// find != 0: (re)build the cluster lists first (they depend on lam and blk only).  rounds: number
// of Cholesky-QR passes over the big clusters (2 = CholeskyQR2: orthogonal to eps for cond(Z_c) < 1e7).
int be_cluster_orth(be_ctx* ctx, const double* lam, const double* tnorm, const int* blk, double* Z, int64_t cnt, int N,
                    int nv, double ctol, int* info, void* scratch, int find, int rounds) {
  ClusterBufs cb;
  cluster_carve((char*)scratch, cnt, N, nv, &cb);
  cudaStream_t st = ctx->stream;
  const int mb = maxbig_of(nv);
  const int tmax = (nv + GT - 1) / GT;
  const int tmaxg = tmax * (tmax + 1) / 2 > mb ? tmax * (tmax + 1) / 2 : mb;
  const int rt = (N + GT - 1) / GT;
  const int tmaxu = (tmax + mb) * rt;   // sum over clusters of ceil(L/64) <= nv/64 + number of clusters
  if (cnt * (int64_t)tmaxu > 0x7fffffffLL) return BE_ERR_SHAPE;
  be_prof_begin(ctx, PK_ORTH);
  if (find) {
    k_find_clusters<<<(unsigned)cnt, 256, 0, st>>>(lam, tnorm, blk, N, nv, ctol, mb, cb);
    LAUNCH_CHECK();
  }
  const size_t sh = (size_t)nv * sizeof(double);
  if (sh > 48 * 1024) BE_CUDA(cudaFuncSetAttribute(k_chol_inv, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sh));
  for (int it = 0; it < rounds; ++it) {
    k_cgram<<<(unsigned)(cnt * tmaxg), 256, 0, st>>>(Z, N, nv, mb, tmaxg, cb);
    LAUNCH_CHECK();
    k_chol_inv<<<(unsigned)(cnt * mb), CHT, sh, st>>>(nv, mb, cb, info);
    LAUNCH_CHECK();
    k_cupdate<<<(unsigned)(cnt * tmaxu), 256, 0, st>>>(Z, N, nv, mb, tmaxu, cb);
    LAUNCH_CHECK();
    k_ccopy<<<(unsigned)(cnt * mb), 256, 0, st>>>(Z, N, nv, mb, cb);
    LAUNCH_CHECK();
  }
  // few matrices: several CTAs per matrix (many: the machine is full anyway, and most CTAs would find nothing to do)
  const int split = cnt * ORTH_SMALL_SPLIT <= 32 * (int64_t)ctx->sm_count ? ORTH_SMALL_SPLIT : 1;
  k_orth_small<<<dim3((unsigned)cnt, (unsigned)split), 256, 0, st>>>(blk, Z, N, nv, cb, info);
  LAUNCH_CHECK();
  be_prof_end(ctx, PK_ORTH, 0.0, 0.0);
  return BE_OK;
}
