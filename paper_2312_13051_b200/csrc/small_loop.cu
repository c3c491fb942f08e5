// Fused Wilson loop for tiny matrices (N <= 8, at most two selected bands): one warp per loop does S1' -> S6 -> S2
// -> S3 -> S4 without writing frames, links or Wilson matrices to memory.
//
//   phase 1  every lane diagonalizes the H(k_j) of its contiguous segment of loop points (one-sided Jacobi,
//            jacobi.cuh), keeps the lowest m eigenvectors; spin resolved: S_red = U^H S U (m x m) is diagonalized
//            in closed form and the frame is rotated into the lower / upper sector.  Frames go to shared memory.
//   phase 2  per sector, every lane multiplies the links M_j = F_j^H F_{j+1} of its segment in order (the closing
//            link uses Phi F_0), then the 32 segment products are combined in order by a shuffle tree
//            (5 steps; a pairwise tree keeps the left-to-right order of PAPER.md:32).
//   phase 3  lane 0: eigenphases of the 1 x 1 / 2 x 2 product in closed form, sorted in (-pi, pi].
// The 2.6 MB grids of configs 1-2 take one launch instead of ~110 (Jacobi, PSO GEMMs, 99 dependent 2 x 2 products).
#include "jacobi.cuh"

namespace {

constexpr int SL_WARPS = 4;   // loops per CTA

struct SmallLoopArgs {
  const cplx* H; GridMap map; int64_t loops; int m;
  const cplx* frames;                      // given frames [loop][n1][m][N] instead of H (nested second level): phase 1 is a copy
  const cplx* close; int phi_at;           // closing phase (or NULL) on the link leaving loop point phi_at
  // plain loop outputs (any may be NULL)
  double* theta; double* absl; double* mingap; cplx* Wout; cplx* X0;
  // spin resolved (S != NULL): sectors of m_lo and m - m_lo vectors
  const void* S; int S_is_diag; int m_lo; double* theta_lo; double* theta_hi; double* pso;
};

__device__ __forceinline__ cplx csqrt_principal(cplx z) {
  const double r = hypot(z.x, z.y);
  if (r == 0.0) return mkc(0.0, 0.0);
  const double a = sqrt(0.5 * (r + fabs(z.x)));
  const double b = 0.5 * z.y / a;
  if (z.x >= 0.0) return mkc(a, b);
  return mkc(fabs(b), copysign(a, z.y));
}

// eigenvalues of the 2 x 2 matrix [[a, b], [c, d]] (the larger one first, the other from the determinant)
__device__ __forceinline__ void eig2x2(cplx a, cplx b, cplx c, cplx d, cplx& l1, cplx& l2) {
  const cplx h = mkc(0.5 * (a.x - d.x), 0.5 * (a.y - d.y));
  const cplx disc = csqrt_principal(cadd(cmul(h, h), cmul(b, c)));
  const cplx mid = mkc(0.5 * (a.x + d.x), 0.5 * (a.y + d.y));
  const cplx p = cadd(mid, disc), q = csub(mid, disc);
  const cplx big = (cabs2(p) >= cabs2(q)) ? p : q;
  const cplx det = csub(cmul(a, d), cmul(b, c));
  l1 = big;
  l2 = (cabs2(big) > 0.0) ? cdiv(det, big) : mkc(0.0, 0.0);
}

__device__ __forceinline__ double angle_pi(cplx l) {
  double t = atan2(l.y, l.x);
  if (t <= -M_PI) t = M_PI;
  return t;
}

// 2 x 2 products, row-major p[0] p[1]; p[2] p[3]; only the leading ms x ms part is meaningful
__device__ __forceinline__ void mul2(cplx (&p)[4], const cplx (&q)[4], int ms) {
  if (ms == 1) { p[0] = cmul(p[0], q[0]); return; }
  cplx r[4];
  r[0] = cmul(p[0], q[0]); cfma(r[0], p[1], q[2]);
  r[1] = cmul(p[0], q[1]); cfma(r[1], p[1], q[3]);
  r[2] = cmul(p[2], q[0]); cfma(r[2], p[3], q[2]);
  r[3] = cmul(p[2], q[1]); cfma(r[3], p[3], q[3]);
  p[0] = r[0]; p[1] = r[1]; p[2] = r[2]; p[3] = r[3];
}

template <int N>
__global__ void __launch_bounds__(SL_WARPS * 32) k_small_loop(const SmallLoopArgs a) {
  extern __shared__ __align__(16) cplx fsm[];   // [warp][sector][point][col 0..1][N]
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int64_t loop = (int64_t)blockIdx.x * SL_WARPS + warp;
  if (loop >= a.loops) return;
  const int n1 = a.map.n1, m = a.m;
  const bool spin = a.S != nullptr;
  const int nsec = spin ? 2 : 1;
  const int msz[2] = {spin ? a.m_lo : m, spin ? m - a.m_lo : 0};
  cplx* F = fsm + (size_t)warp * 2 * n1 * 2 * N;
  const int seg = (n1 + 31) / 32;
  const int j0 = lane * seg, j1 = (j0 + seg < n1) ? j0 + seg : n1;
  double gap = INFINITY;
  // ---- phase 1
  for (int j = j0; j < j1; ++j) {
    if (a.frames) {
      for (int k = 0; k < m; ++k)
#pragma unroll
        for (int r = 0; r < N; ++r) F[((size_t)j * 2 + k) * N + r] = a.frames[((loop * n1 + j) * m + k) * N + r];
      continue;
    }
    const int64_t src = gridmap_index(a.map, loop, j);
    cplx V[N][N];
    double ev[N];
    int ord[N];
    jacobi_hermitian<N>(a.H + src * (N * N), ev, V, ord);
    cplx U[2][N];
    double e[3] = {0.0, 0.0, 0.0};
#pragma unroll
    for (int c = 0; c < N; ++c) {
      double nn = 0.0;
#pragma unroll
      for (int r = 0; r < N; ++r) nn += cabs2(V[c][r]);
      const double sc = 1.0 / sqrt(nn);
#pragma unroll
      for (int k = 0; k < 3; ++k) if (k < N && ord[k] == c) e[k] = ev[c];
#pragma unroll
      for (int k = 0; k < 2; ++k)
        if (k < N && ord[k] == c) {
#pragma unroll
          for (int r = 0; r < N; ++r) U[k][r] = cscale(sc, V[c][r]);
        }
    }
    if (m < N) gap = fmin(gap, e[m] - e[m - 1]);
    if (a.X0 && j == 0) {
      for (int k = 0; k < m; ++k)
#pragma unroll
        for (int r = 0; r < N; ++r) a.X0[(loop * m + k) * N + r] = U[k][r];
    }
    if (!spin) {
      for (int k = 0; k < m; ++k)
#pragma unroll
        for (int r = 0; r < N; ++r) F[((size_t)j * 2 + k) * N + r] = U[k][r];
      continue;
    }
    // S_red = U^H S U (m x m Hermitian, m <= 2)
    cplx SU[2][N];
    for (int k = 0; k < m; ++k)
#pragma unroll
      for (int r = 0; r < N; ++r) {
        if (a.S_is_diag) SU[k][r] = cscale(((const double*)a.S)[r], U[k][r]);
        else {
          cplx t = mkc(0.0, 0.0);
#pragma unroll
          for (int c = 0; c < N; ++c) cfma(t, ((const cplx*)a.S)[r * N + c], U[k][c]);
          SU[k][r] = t;
        }
      }
    double s00 = 0.0, s11 = 0.0;
    cplx s01 = mkc(0.0, 0.0);
#pragma unroll
    for (int r = 0; r < N; ++r) {
      s00 += U[0][r].x * SU[0][r].x + U[0][r].y * SU[0][r].y;
      if (m == 2) { s11 += U[1][r].x * SU[1][r].x + U[1][r].y * SU[1][r].y; cfmac(s01, U[0][r], SU[1][r]); }
    }
    // eigenvectors of [[s00, s01], [conj(s01), s11]]: columns (c, -s conj(ph)), (s ph, c) ... as a rotation
    cplx R[2][2] = {{mkc(1.0, 0.0), mkc(0.0, 0.0)}, {mkc(0.0, 0.0), mkc(1.0, 0.0)}};   // R[col][row]
    double sig[2] = {s00, s11};
    if (m == 2) {
      const double ab = sqrt(cabs2(s01));
      if (ab > 0.0) {
        const double zeta = (s11 - s00) / (2.0 * ab);
        const double t = copysign(1.0, zeta) / (fabs(zeta) + sqrt(1.0 + zeta * zeta));
        const double cs = 1.0 / sqrt(1.0 + t * t), sn = cs * t;
        const cplx ph = mkc(s01.x / ab, s01.y / ab);          // s01 = |s01| ph
        // v0 = (cs, -sn conj(ph)), v1 = (sn ph, cs): eigenvalues s00 - t |s01|, s11 + t |s01|
        R[0][0] = mkc(cs, 0.0); R[0][1] = mkc(-sn * ph.x, sn * ph.y);
        R[1][0] = mkc(sn * ph.x, sn * ph.y); R[1][1] = mkc(cs, 0.0);
        sig[0] = s00 - t * ab; sig[1] = s11 + t * ab;
      }
      if (sig[1] < sig[0]) {
        const double ts = sig[0]; sig[0] = sig[1]; sig[1] = ts;
        const cplx t0 = R[0][0], t1 = R[0][1];
        R[0][0] = R[1][0]; R[0][1] = R[1][1]; R[1][0] = t0; R[1][1] = t1;
      }
    }
    if (a.pso) for (int k = 0; k < m; ++k) a.pso[(loop * n1 + j) * m + k] = sig[k];
    // sector frames: column k of U R, k < m_lo lower sector, the rest upper
    for (int k = 0; k < m; ++k) {
      const int sec = (k < a.m_lo) ? 0 : 1, kk = (k < a.m_lo) ? k : k - a.m_lo;
#pragma unroll
      for (int r = 0; r < N; ++r) {
        cplx t = cmul(U[0][r], R[k][0]);
        if (m == 2) cfma(t, U[1][r], R[k][1]);
        F[(((size_t)sec * n1 + j) * 2 + kk) * N + r] = t;
      }
    }
  }
  __syncwarp();
  if (a.mingap) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) gap = fmin(gap, __shfl_xor_sync(0xffffffffu, gap, o));
    if (lane == 0) a.mingap[loop] = gap;
  }
  // ---- phases 2, 3 per sector
  for (int sec = 0; sec < nsec; ++sec) {
    const int ms = msz[sec];
    if (ms == 0) continue;
    const cplx* Fs = F + (size_t)sec * n1 * 2 * N;
    cplx P[4] = {mkc(1.0, 0.0), mkc(0.0, 0.0), mkc(0.0, 0.0), mkc(1.0, 0.0)};
    for (int j = j0; j < j1; ++j) {
      const int jn = (j + 1 == n1) ? 0 : j + 1;
      const bool ph = a.close && j == a.phi_at;
      cplx M[4] = {mkc(0.0, 0.0), mkc(0.0, 0.0), mkc(0.0, 0.0), mkc(0.0, 0.0)};
      for (int x = 0; x < ms; ++x)
        for (int y = 0; y < ms; ++y) {
          cplx t = mkc(0.0, 0.0);
#pragma unroll
          for (int r = 0; r < N; ++r) {
            cplx b = Fs[((size_t)jn * 2 + y) * N + r];
            if (ph) b = cmul(a.close[r], b);
            cfmac(t, Fs[((size_t)j * 2 + x) * N + r], b);
          }
          M[x * 2 + y] = t;
        }
      mul2(P, M, ms);
    }
    // ordered combination of the 32 segment products: P_lane <- P_lane P_{lane + off}
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
      cplx Q[4];
#pragma unroll
      for (int e = 0; e < 4; ++e)
        Q[e] = mkc(__shfl_down_sync(0xffffffffu, P[e].x, off), __shfl_down_sync(0xffffffffu, P[e].y, off));
      if ((lane & (2 * off - 1)) == 0) mul2(P, Q, ms);
    }
    if (lane != 0) continue;
    if (a.Wout && !spin) {   // column-major m x m, as be_chain_product writes it
      for (int x = 0; x < ms; ++x) for (int y = 0; y < ms; ++y) a.Wout[loop * ms * ms + y * ms + x] = P[x * 2 + y];
    }
    double* th = spin ? (sec == 0 ? a.theta_lo : a.theta_hi) : a.theta;
    double* ab = spin ? nullptr : a.absl;
    if (ms == 1) {
      if (th) th[loop] = angle_pi(P[0]);
      if (ab) ab[loop] = sqrt(cabs2(P[0]));
    } else {
      cplx l1, l2;
      eig2x2(P[0], P[1], P[2], P[3], l1, l2);
      const double t1 = angle_pi(l1), t2 = angle_pi(l2);
      const bool sw = t2 < t1;
      if (th) { th[loop * 2] = sw ? t2 : t1; th[loop * 2 + 1] = sw ? t1 : t2; }
      if (ab) { ab[loop * 2] = sqrt(cabs2(sw ? l2 : l1)); ab[loop * 2 + 1] = sqrt(cabs2(sw ? l1 : l2)); }
    }
  }
}

}  // namespace

// Whether the fused kernel covers a call (N <= 8, m <= 2, frames of a loop fit shared memory).
bool be_small_loop_applies(int N, int m, int n1) {
  return N >= 1 && N <= 8 && m >= 1 && m <= 2 && m <= N &&
         (size_t)SL_WARPS * 2 * n1 * 2 * N * sizeof(cplx) <= 200 * 1024;
}

int be_small_loop(be_ctx* ctx, const cplx* H, const cplx* frames, const GridMap& map, int N, int m, const cplx* d_close, int phi_at,
                  double* d_theta, double* d_abs, double* d_mingap, cplx* Wout, cplx* X0, const void* dS, int S_is_diag,
                  int m_lo, double* d_theta_lo, double* d_theta_hi, double* d_pso) {
  if (!be_small_loop_applies(N, m, map.n1)) return BE_ERR_UNSUPPORTED;
  SmallLoopArgs a;
  a.H = H; a.frames = frames; a.map = map; a.loops = map.loops; a.m = m; a.close = d_close; a.phi_at = phi_at;
  a.theta = d_theta; a.absl = d_abs; a.mingap = d_mingap; a.Wout = Wout; a.X0 = X0;
  a.S = dS; a.S_is_diag = S_is_diag; a.m_lo = m_lo; a.theta_lo = d_theta_lo; a.theta_hi = d_theta_hi; a.pso = d_pso;
  const size_t smem = (size_t)SL_WARPS * 2 * map.n1 * 2 * N * sizeof(cplx);
  const unsigned blocks = (unsigned)((map.loops + SL_WARPS - 1) / SL_WARPS);
  be_prof_begin(ctx, PK_JACOBI);
  switch (N) {
#define CASE(n) case n: \
    if (smem > 48 * 1024) BE_CUDA(cudaFuncSetAttribute(k_small_loop<n>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)); \
    k_small_loop<n><<<blocks, SL_WARPS * 32, smem, ctx->stream>>>(a); break;
    CASE(1) CASE(2) CASE(3) CASE(4) CASE(5) CASE(6) CASE(7) CASE(8)
#undef CASE
    default: return BE_ERR_UNSUPPORTED;
  }
  be_prof_end(ctx, PK_JACOBI, (double)map.loops * map.n1 * N * N * 16.0, (double)map.loops * map.n1 * 8.0 * N * m * m);
  ctx->launches++;
  return (int)cudaGetLastError();
}
