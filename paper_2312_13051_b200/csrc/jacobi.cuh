// Cyclic one-sided (Hestenes) Jacobi for one Hermitian N x N matrix held by one thread, N <= 8 (S1').
// Shared by the batched kernel (eigh_small.cu) and the fused tiny-N loop kernel (small_loop.cu).
//
// One-sided Jacobi orthogonalizes the columns of G = A V.  Applied to H itself it fails on the
// chiral / particle-hole symmetric spectra of the paper's toy models (BHZ Eq. 7, BBH: E = +-eps
// doubly degenerate makes H^H H proportional to 1, so the columns are orthogonal from the start
// and no eigenvector information is produced).  It is therefore applied to the positive definite
// shift A = H + s 1, s = 1.5 ||H||_F: singular values of A are lambda + s and V holds the
// eigenvectors.  Absolute accuracy eps (s + ||H||) <= 3 eps ||H||_F.
#pragma once
#include "be_common.cuh"
#include <float.h>

// h: row-major Hermitian input, upper triangle read.  On return ev[j] (unsorted) and V[j][.] (column j,
// unnormalised up to rounding) are eigenpairs, ord[] lists the columns by ascending eigenvalue.
template <int N>
__device__ __forceinline__ bool jacobi_hermitian(const cplx* __restrict__ h, double (&ev)[N], cplx (&V)[N][N], int (&ord)[N]) {
  cplx G[N][N];   // [column][row]
  double fro = 0.0;
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
  return done;
}
