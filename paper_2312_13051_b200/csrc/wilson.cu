// S2-S7 -- link overlaps, ordered Wilson product, spin-resolved and nested variants, invariants.
// The contractions are DMMA ZGEMMs (zgemm.cu); this file holds the small glue kernels and the
// host-side sequencing of one chunk of loops.
#include "be_common.cuh"
#include <float.h>

namespace {

// min over the loop of the gaps at the edges of the band window [lo, hi): E[hi] - E[hi-1] (R8) and,
// for lo > 0, E[lo] - E[lo-1]; +inf when the window has no edge inside the spectrum.
__global__ void k_mingap(const double* __restrict__ E, int N, int lo, int hi, int n1, int64_t loops,
                         double* __restrict__ out) {
  const int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (l >= loops) return;
  double g = INFINITY;
  for (int j = 0; j < n1; ++j) {
    const double* e = E + (l * n1 + j) * (int64_t)N;
    if (hi < N) g = fmin(g, e[hi] - e[hi - 1]);
    if (lo > 0) g = fmin(g, e[lo] - e[lo - 1]);
  }
  out[l] = g;
}

// bad[l] |= any eigensolve of loop l was flagged (info != 0) or returned a non-finite lowest eigenvalue
__global__ void k_flag_loops(const int* __restrict__ info, const double* __restrict__ E, int ldE, int n1, int64_t nl,
                             int* __restrict__ bad0, int* __restrict__ bad1) {
  const int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (l >= nl) return;
  int f = 0;
  for (int j = 0; j < n1; ++j) {
    const int64_t c = l * n1 + j;
    if (info[c]) f = 1;
    if (E && !isfinite(E[c * ldE])) f = 1;
  }
  if (f) { bad0[l] = 1; if (bad1) bad1[l] = 1; }
}

// SX[c][v][r] = S[r] * X[c][v][r] for a real diagonal S.
__global__ void k_scale_rows(const cplx* __restrict__ X, const double* __restrict__ S,
                             cplx* __restrict__ SX, int N, int64_t total) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= total) return;
  const double s = S[i % N];
  const cplx x = X[i];
  SX[i] = mkc(s * x.x, s * x.y);
}

// Winding of Theta_i = sum_n theta_n around a closed cycle (Eq. 6); one warp per cycle.
__global__ void k_winding(const double* __restrict__ theta, int64_t n_cycles, int n_points, int m,
                          double* __restrict__ wind) {
  const int64_t cyc = blockIdx.x;
  const int lane = threadIdx.x;
  const double* th = theta + cyc * (int64_t)n_points * m;
  double acc = 0.0;
  for (int i = lane; i < n_points; i += 32) {
    const int i2 = (i + 1 == n_points) ? 0 : i + 1;
    double a = 0.0, b = 0.0;
    for (int n = 0; n < m; ++n) { a += th[(int64_t)i * m + n]; b += th[(int64_t)i2 * m + n]; }
    double d = fmod(b - a + M_PI, 2.0 * M_PI);
    if (d < 0.0) d += 2.0 * M_PI;
    d -= M_PI;
    if (d <= -M_PI) d = M_PI;
    acc += d;
  }
  acc = warp_sum(acc);
  if (lane == 0) wind[cyc] = acc / (2.0 * M_PI);
}

__device__ __forceinline__ cplx csqrt2(cplx z) {
  const double r = hypot(z.x, z.y);
  if (r == 0.0) return mkc(0.0, 0.0);
  const double a = sqrt(0.5 * (r + fabs(z.x)));
  const double b = 0.5 * z.y / a;
  if (z.x >= 0.0) return mkc(a, b);
  return mkc(fabs(b), copysign(a, z.y));
}

__device__ __forceinline__ double branch_angle(cplx l, double cut) {
  double t = atan2(l.y, l.x);
  if (t > cut) t -= 2.0 * M_PI;
  if (t <= cut - 2.0 * M_PI) t += 2.0 * M_PI;
  return t;
}

// Nested loop, m <= 2 (closed form): per first-level Wilson matrix W (column-major m x m) the
// sorted phases on (-pi, pi] and the orthonormalized right eigenvectors of the Wannier bands
// wb_lo..wb_hi-1 ranked on the branch (cut - 2 pi, cut] (R9).  Vs: [loop][ns][m] column-major.
__global__ void k_nested_select_small(const cplx* __restrict__ W, int64_t cnt, int m, int wb_lo,
                                      int wb_hi, double cut, double* __restrict__ theta1,
                                      cplx* __restrict__ Vs) {
  const int64_t c = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (c >= cnt) return;
  const int ns = wb_hi - wb_lo;
  if (m == 1) {
    double t = atan2(W[c].y, W[c].x);
    if (t <= -M_PI) t = M_PI;
    theta1[c] = t;
    if (ns == 1) Vs[c] = mkc(1.0, 0.0);
    return;
  }
  const cplx a = W[c * 4], cc = W[c * 4 + 1], b = W[c * 4 + 2], d = W[c * 4 + 3];
  const cplx h = mkc(0.5 * (a.x - d.x), 0.5 * (a.y - d.y));
  const cplx disc = csqrt2(cadd(cmul(h, h), cmul(b, cc)));
  const cplx mid = mkc(0.5 * (a.x + d.x), 0.5 * (a.y + d.y));
  const cplx p = cadd(mid, disc), q = csub(mid, disc);
  const cplx big = (cabs2(p) >= cabs2(q)) ? p : q;
  const cplx det = csub(cmul(a, d), cmul(b, cc));
  cplx lam[2];
  lam[0] = big;
  lam[1] = (cabs2(big) > 0.0) ? cdiv(det, big) : mkc(0.0, 0.0);
  double t0 = atan2(lam[0].y, lam[0].x), t1 = atan2(lam[1].y, lam[1].x);
  if (t0 <= -M_PI) t0 = M_PI;
  if (t1 <= -M_PI) t1 = M_PI;
  theta1[c * 2] = fmin(t0, t1);
  theta1[c * 2 + 1] = fmax(t0, t1);
  const double b0 = branch_angle(lam[0], cut), b1 = branch_angle(lam[1], cut);
  int order[2];
  if (b0 <= b1) { order[0] = 0; order[1] = 1; } else { order[0] = 1; order[1] = 0; }
  cplx vecs[2][2];
  for (int s = 0; s < ns; ++s) {
    const cplx l = lam[order[wb_lo + s]];
    // (W - l) v = 0: candidates (b, l - a) and (l - d, c); take the better conditioned one
    const cplx v1a = b, v1b = csub(l, a);
    const cplx v2a = csub(l, d), v2b = cc;
    const double n1 = cabs2(v1a) + cabs2(v1b), n2 = cabs2(v2a) + cabs2(v2b);
    cplx va, vb;
    if (n1 >= n2) { va = v1a; vb = v1b; } else { va = v2a; vb = v2b; }
    double nn = fmax(n1, n2);
    if (nn == 0.0) { va = mkc(s == 0 ? 1.0 : 0.0, 0.0); vb = mkc(s == 0 ? 0.0 : 1.0, 0.0); nn = 1.0; }
    const double sc = 1.0 / sqrt(nn);
    vecs[s][0] = cscale(sc, va); vecs[s][1] = cscale(sc, vb);
  }
  if (ns == 2) {   // Gram-Schmidt (the span is the whole space)
    cplx dot = mkc(0.0, 0.0);
    cfmac(dot, vecs[0][0], vecs[1][0]); cfmac(dot, vecs[0][1], vecs[1][1]);
    cfms(vecs[1][0], dot, vecs[0][0]); cfms(vecs[1][1], dot, vecs[0][1]);
    const double nn = cabs2(vecs[1][0]) + cabs2(vecs[1][1]);
    const double sc = nn > 0.0 ? 1.0 / sqrt(nn) : 0.0;
    vecs[1][0] = cscale(sc, vecs[1][0]); vecs[1][1] = cscale(sc, vecs[1][1]);
  }
  for (int s = 0; s < ns; ++s) { Vs[(c * ns + s) * 2] = vecs[s][0]; Vs[(c * ns + s) * 2 + 1] = vecs[s][1]; }
}

}  // namespace

#define LAUNCH_CHECK() do { ctx->launches++; cudaError_t e__ = cudaGetLastError(); if (e__ != cudaSuccess) return (int)e__; } while (0)

int be_mingap(be_ctx* ctx, const double* E, int N, int lo, int hi, int n1, int64_t loops, double* out) {
  k_mingap<<<(unsigned)((loops + 127) / 128), 128, 0, ctx->stream>>>(E, N, lo, hi, n1, loops, out);
  LAUNCH_CHECK();
  return BE_OK;
}

int be_flag_loops(be_ctx* ctx, const int* info, const double* E, int ldE, int n1, int64_t nl, int* bad0, int* bad1) {
  k_flag_loops<<<(unsigned)((nl + 127) / 128), 128, 0, ctx->stream>>>(info, E, ldE, n1, nl, bad0, bad1);
  LAUNCH_CHECK();
  return BE_OK;
}

// Diagonal S with a dominant value b:  U^H S U = b I + U_A^H (S_A - b) U_A, where A is the set of rows with
// S[r] != b (U^H U = I).  XA[c][v][i] = X[c][v][sel[i]], SXA = (S[sel[i]] - b) XA; leading dimension nsel.
__global__ void k_pack_rows(const cplx* __restrict__ X, const double* __restrict__ S, const int* __restrict__ sel,
                            double b, cplx* __restrict__ XA, cplx* __restrict__ SXA, int N, int nsel, int64_t total) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= total) return;
  const int64_t col = i / nsel;
  const int r = sel[i - col * nsel];
  const double s = S[r] - b;
  const cplx x = X[col * N + r];
  XA[i] = x;
  SXA[i] = mkc(s * x.x, s * x.y);
}

__global__ void k_add_diag(cplx* __restrict__ A, int m, int64_t total, double b) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= total) return;
  const int64_t c = i / m;
  const int k = (int)(i - c * m);
  A[c * (int64_t)m * m + (int64_t)k * m + k].x += b;
}

int be_pack_rows(be_ctx* ctx, const cplx* X, const double* S, const int* sel, double b, cplx* XA, cplx* SXA, int N,
                 int nsel, int64_t cols) {
  const int64_t total = cols * nsel;
  if (total == 0) return BE_OK;
  k_pack_rows<<<(unsigned)((total + 255) / 256), 256, 0, ctx->stream>>>(X, S, sel, b, XA, SXA, N, nsel, total);
  LAUNCH_CHECK();
  return BE_OK;
}

int be_add_diag(be_ctx* ctx, cplx* A, int m, int64_t cnt, double b) {
  const int64_t total = cnt * m;
  k_add_diag<<<(unsigned)((total + 255) / 256), 256, 0, ctx->stream>>>(A, m, total, b);
  LAUNCH_CHECK();
  return BE_OK;
}

int be_scale_rows(be_ctx* ctx, const cplx* X, const double* S, cplx* SX, int N, int64_t total) {
  k_scale_rows<<<(unsigned)((total + 255) / 256), 256, 0, ctx->stream>>>(X, S, SX, N, total);
  LAUNCH_CHECK();
  return BE_OK;
}

int be_winding_impl(be_ctx* ctx, const double* theta, int64_t n_cycles, int n_points, int m, double* wind) {
  k_winding<<<(unsigned)n_cycles, 32, 0, ctx->stream>>>(theta, n_cycles, n_points, m, wind);
  LAUNCH_CHECK();
  return BE_OK;
}

int be_nested_select_small(be_ctx* ctx, const cplx* W, int64_t cnt, int m, int wb_lo, int wb_hi,
                           double cut, double* theta1, cplx* Vs) {
  k_nested_select_small<<<(unsigned)((cnt + 127) / 128), 128, 0, ctx->stream>>>(W, cnt, m, wb_lo, wb_hi, cut, theta1, Vs);
  LAUNCH_CHECK();
  return BE_OK;
}

// Chain of one chunk: frames F [outer][inner][m][N] (column-major N x m each, ld N) ->
// links M_j = F_j^H F_{j+1} (ring, Phi on the link at inner index phi_at) -> ordered product
// W = M_0 M_1 ... M_{n1-1} per outer.  The product is a pairwise tree, P_j <- P_2j P_2j+1 level by level
// (ceil(log2 n1) batched GEMM launches instead of n1 - 1 dependent ones; an odd last factor is carried
// over): PAPER.md:32, 36-38 fix the ORDER of the factors, which a tree of adjacent pairs keeps.
// Returns W (column-major m x m, stride m*m) in *Wout; when Wdst is not NULL the final product is written
// there (a buffer that outlives the chunk).
int be_chain_product(be_ctx* ctx, const cplx* F, int N, int m, int64_t outer, int n1,
                     const cplx* d_close, int phi_at, cplx* Wdst, cplx** Wout) {
  const int64_t mm = (int64_t)m * m;
  const int half = (n1 + 1) / 2;
  cplx* M = (cplx*)be_arena_alloc(ctx, (size_t)outer * n1 * mm * sizeof(cplx));
  cplx* W0 = (cplx*)be_arena_alloc(ctx, (size_t)outer * half * mm * sizeof(cplx));
  cplx* W1 = (cplx*)be_arena_alloc(ctx, (size_t)outer * ((half + 1) / 2) * mm * sizeof(cplx));
  if (!M || !W0 || !W1) return BE_ERR_NOMEM;
  ZgemmParams g;
  g.M = m; g.N = m; g.K = N;
  g.A = F; g.lda = N; g.sAi = (int64_t)N * m; g.sAo = (int64_t)n1 * N * m;
  g.B = F; g.ldb = N; g.sBi = (int64_t)N * m; g.sBo = (int64_t)n1 * N * m;
  g.C = M; g.ldc = m; g.sCi = mm; g.sCo = (int64_t)n1 * mm;
  g.inner = n1; g.batch = outer * n1;
  g.ringB = 1; g.phiB = d_close; g.phi_at = phi_at;
  g.alpha = mkc(1.0, 0.0); g.beta = mkc(0.0, 0.0); g.lower = 0;
  g.A2 = nullptr; g.B2 = nullptr; g.sA2o = g.sB2o = 0; g.ksplit = 0;
  BE_TRY(be_zgemm(ctx, BE_OP_C, BE_OP_N, g));
  if (n1 == 1) {
    cplx* dst = Wdst ? Wdst : W0;
    BE_CUDA(cudaMemcpyAsync(dst, M, (size_t)outer * mm * sizeof(cplx), cudaMemcpyDeviceToDevice, ctx->stream));
    *Wout = dst;
    return BE_OK;
  }
  const cplx* cur = M;            // cnt factors per loop, contiguous: cur[o][j]
  int cnt = n1, level = 0;
  cplx* bufs[2] = {W0, W1};
  while (cnt > 1) {
    const int pairs = cnt / 2, ncnt = pairs + (cnt & 1);
    cplx* dst = (ncnt == 1 && Wdst) ? Wdst : bufs[level & 1];
    ZgemmParams p = zgemm_simple(m, m, m, cur, m, (int64_t)cnt * mm, cur + mm, m, (int64_t)cnt * mm,
                                 dst, m, (int64_t)ncnt * mm, (int64_t)outer * pairs);
    p.sAi = 2 * mm; p.sBi = 2 * mm; p.sCi = mm; p.inner = pairs;
    BE_TRY(be_zgemm(ctx, BE_OP_N, BE_OP_N, p));
    if (cnt & 1)   // the unpaired last factor moves up unchanged
      BE_CUDA(cudaMemcpy2DAsync(dst + (int64_t)pairs * mm, (size_t)ncnt * mm * sizeof(cplx), cur + (int64_t)(cnt - 1) * mm,
                                (size_t)cnt * mm * sizeof(cplx), (size_t)mm * sizeof(cplx), (size_t)outer,
                                cudaMemcpyDeviceToDevice, ctx->stream));
    cur = dst; cnt = ncnt; ++level;
  }
  *Wout = (cplx*)cur;
  return BE_OK;
}
