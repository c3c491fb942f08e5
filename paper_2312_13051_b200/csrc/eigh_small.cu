// S1' -- many-small-matrix regime (N <= 8): cyclic one-sided (Hestenes) Jacobi, one thread per
// matrix, everything in registers / local memory.
//
// One-sided Jacobi orthogonalizes the columns of G = A V.  Applied to H itself it fails on the
// chiral / particle-hole symmetric spectra of the paper's toy models (BHZ Eq. 7, BBH: E = +-eps
// doubly degenerate makes H^H H proportional to 1, so the columns are orthogonal from the start
// and no eigenvector information is produced).  It is therefore applied to the positive definite
// shift A = H + s 1, s = 1.5 ||H||_F: singular values of A are lambda + s and V holds the
// eigenvectors.  Absolute accuracy eps (s + ||H||) <= 3 eps ||H||_F.
#include "be_common.cuh"
#include <float.h>

namespace {

template <int N>
__global__ void __launch_bounds__(128) k_jacobi(const cplx* __restrict__ H, GridMap map, int64_t loop0,
                                                int64_t cnt, int nv, double* __restrict__ E,
                                                cplx* __restrict__ X, int* __restrict__ info) {
  const int64_t c = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (c >= cnt) return;
  const int64_t src = gridmap_index(map, loop0 + c / map.n1, (int)(c % map.n1));
  const cplx* h = H + src * (N * N);
  cplx G[N][N], V[N][N];   // [column][row]
  double fro = 0.0;
  // column j of the Hermitian matrix from the upper triangle of the row-major input:
  // A[r][j] = H[r][j] for r <= j, conj(H[j][r]) for r > j
#pragma unroll
  for (int j = 0; j < N; ++j)
#pragma unroll
    for (int r = 0; r < N; ++r) {
      cplx a = (r <= j) ? h[r * N + j] : cconj(h[j * N + r]);
      if (r == j) a.y = 0.0;
      G[j][r] = a;
      fro += cabs2(a);
      V[j][r] = mkc(r == j ? 1.0 : 0.0, 0.0);
    }
  const double s = 1.5 * sqrt(fro) + DBL_MIN;
#pragma unroll
  for (int j = 0; j < N; ++j) G[j][j].x += s;

  int sweeps = 0;
  bool done = (N == 1);
  while (!done && sweeps < 40) {
    done = true;
    ++sweeps;
#pragma unroll
    for (int p = 0; p < N - 1; ++p)
#pragma unroll
      for (int q = p + 1; q < N; ++q) {
        double al = 0.0, be = 0.0;
        cplx ga = mkc(0.0, 0.0);
#pragma unroll
        for (int r = 0; r < N; ++r) {
          al += cabs2(G[p][r]); be += cabs2(G[q][r]);
          cfmac(ga, G[p][r], G[q][r]);
        }
        const double ag = sqrt(cabs2(ga));
        if (ag > 1e-15 * sqrt(al * be) && ag > 0.0) {
          done = false;
          const double zeta = (be - al) / (2.0 * ag);
          const double t = copysign(1.0, zeta) / (fabs(zeta) + sqrt(1.0 + zeta * zeta));
          const double cs = 1.0 / sqrt(1.0 + t * t), sn = cs * t;
          // g_q~ = e^{-i theta} g_q with gamma = |gamma| e^{i theta}
          const cplx ph = mkc(ga.x / ag, -ga.y / ag);
#pragma unroll
          for (int r = 0; r < N; ++r) {
            const cplx gp = G[p][r], gq = cmul(ph, G[q][r]);
            G[p][r] = mkc(cs * gp.x - sn * gq.x, cs * gp.y - sn * gq.y);
            G[q][r] = mkc(sn * gp.x + cs * gq.x, sn * gp.y + cs * gq.y);
            const cplx vp = V[p][r], vq = cmul(ph, V[q][r]);
            V[p][r] = mkc(cs * vp.x - sn * vq.x, cs * vp.y - sn * vq.y);
            V[q][r] = mkc(sn * vp.x + cs * vq.x, sn * vp.y + cs * vq.y);
          }
        }
      }
  }
  if (info) info[c] = done ? 0 : 1;
  double ev[N];
  int ord[N];
#pragma unroll
  for (int j = 0; j < N; ++j) {
    double nn = 0.0;
#pragma unroll
    for (int r = 0; r < N; ++r) nn += cabs2(G[j][r]);
    ev[j] = sqrt(nn) - s;
    ord[j] = j;
  }
  // insertion sort (ascending)
#pragma unroll
  for (int a = 1; a < N; ++a)
#pragma unroll
    for (int b = a; b > 0; --b)
      if (ev[ord[b]] < ev[ord[b - 1]]) { const int tmp = ord[b]; ord[b] = ord[b - 1]; ord[b - 1] = tmp; }
#pragma unroll
  for (int j = 0; j < N; ++j) {
    double val = 0.0;
#pragma unroll
    for (int a = 0; a < N; ++a) if (ord[j] == a) val = ev[a];
    E[c * N + j] = val;
  }
  if (X) {
#pragma unroll
    for (int j = 0; j < N; ++j) {
      if (j < nv) {
#pragma unroll
        for (int a = 0; a < N; ++a)
          if (ord[j] == a) {
            // normalise (V is unitary up to rounding; re-normalise the column)
            double nn = 0.0;
#pragma unroll
            for (int r = 0; r < N; ++r) nn += cabs2(V[a][r]);
            const double sc = 1.0 / sqrt(nn);
#pragma unroll
            for (int r = 0; r < N; ++r) X[c * (int64_t)(N * nv) + j * N + r] = cscale(sc, V[a][r]);
          }
      }
    }
  }
}

}  // namespace

int be_eigh_small(be_ctx* ctx, const cplx* H, const GridMap& map, int64_t loop0, int64_t cnt, int N,
                  int nv, double* E, cplx* X, int* info) {
  const unsigned blocks = (unsigned)((cnt + 127) / 128);
  cudaStream_t st = ctx->stream;
  be_prof_begin(ctx, PK_JACOBI);
  switch (N) {
#define CASE(n) case n: k_jacobi<n><<<blocks, 128, 0, st>>>(H, map, loop0, cnt, nv, E, X, info); break;
    CASE(1) CASE(2) CASE(3) CASE(4) CASE(5) CASE(6) CASE(7) CASE(8)
#undef CASE
    default: return BE_ERR_UNSUPPORTED;
  }
  be_prof_end(ctx, PK_JACOBI, (double)cnt * N * (N + (double)nv + 1) * 16.0, 0.0);
  ctx->launches++;
  return (int)cudaGetLastError();
}
