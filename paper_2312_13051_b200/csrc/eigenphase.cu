// S4 -- eigenphases theta_n = arg lambda_n(W) of the Wilson matrices (Eq. 2,
// PAPER.md:127 Eq. 8 "Im Ln").  W is NOT unitary at finite Delta k and is not unitarized (R4), so
// this is a general complex eigenvalue problem:
//   m = 1, 2 : closed form, one thread per matrix
//   m > 2    : Householder reduction to Hessenberg form, then explicit single-shift complex QR on
//              the active window (eigenvalues only), one CTA per matrix, W resident in L2.
// Output sorted ascending on the branch (-pi, pi] (R7) by a rank sort.
#include "be_common.cuh"
#include <float.h>
#include <cooperative_groups.h>

namespace {

__device__ __forceinline__ cplx csqrt_(cplx z) {
  const double r = hypot(z.x, z.y);
  if (r == 0.0) return mkc(0.0, 0.0);
  double a = sqrt(0.5 * (r + fabs(z.x)));
  double b = 0.5 * z.y / a;
  if (z.x >= 0.0) return mkc(a, b);
  return mkc(fabs(b), copysign(a, z.y));
}

// eigenvalues of [[a, b], [c, d]]
__device__ __forceinline__ void eig2(cplx a, cplx b, cplx c, cplx d, cplx& l1, cplx& l2) {
  const cplx h = mkc(0.5 * (a.x - d.x), 0.5 * (a.y - d.y));
  const cplx disc = csqrt_(cadd(cmul(h, h), cmul(b, c)));
  const cplx mid = mkc(0.5 * (a.x + d.x), 0.5 * (a.y + d.y));
  // larger-modulus root first, the other from the determinant (avoids cancellation)
  const cplx p = cadd(mid, disc), q = csub(mid, disc);
  const cplx big = (cabs2(p) >= cabs2(q)) ? p : q;
  const cplx det = csub(cmul(a, d), cmul(b, c));
  l1 = big;
  l2 = (cabs2(big) > 0.0) ? cdiv(det, big) : mkc(0.0, 0.0);
}

__global__ void k_eig_small(const cplx* __restrict__ W, int64_t cnt, int m, cplx* __restrict__ lam) {
  const int64_t c = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (c >= cnt) return;
  if (m == 1) { lam[c] = W[c]; return; }
  const cplx* w = W + c * 4;   // column-major 2x2: w[0]=a, w[1]=c, w[2]=b, w[3]=d
  cplx l1, l2;
  eig2(w[0], w[2], w[1], w[3], l1, l2);
  lam[c * 2] = l1; lam[c * 2 + 1] = l2;
}

// ------------------------------------------------------------------------------------------
// Householder reduction to upper Hessenberg form, one CTA of 1024 threads per matrix (there are few
// Wilson matrices -- 48 at the bench workload -- so the per-matrix latency is what counts).
//   left  update: warp per pair of columns (dot over rows with lanes, then axpy)
//   right update: thread = (row i, column slice s of 2); partial y = H v per slice through shared memory
template <int HESS_THREADS>
__global__ void __launch_bounds__(HESS_THREADS) k_hessenberg(cplx* __restrict__ W, int m) {
  extern __shared__ cplx vsh[];   // v[m], y[2][m]
  __shared__ double redd[33];
  __shared__ cplx sh_alpha;
  cplx* v = vsh; cplx* y = vsh + m;
  cplx* H = W + blockIdx.x * (int64_t)m * m;
  const int tid = threadIdx.x, nt = HESS_THREADS, warp = tid >> 5, lane = tid & 31, nw = nt >> 5;
  for (int k = 0; k < m - 2; ++k) {
    double ss = 0.0;
    for (int r = k + 1 + tid; r < m; r += nt) {
      const cplx x = H[r + (int64_t)k * m];
      if (r == k + 1) sh_alpha = x; else ss += cabs2(x);
    }
    const double xn2 = block_sum(ss, redd);
    const cplx alpha = sh_alpha;
    if (xn2 == 0.0 && alpha.y == 0.0) { __syncthreads(); continue; }
    const double beta = -copysign(sqrt(cabs2(alpha) + xn2), alpha.x);
    const cplx tau = mkc((beta - alpha.x) / beta, -alpha.y / beta);
    const cplx scale = cdiv(mkc(1.0, 0.0), mkc(alpha.x - beta, alpha.y));
    for (int r = k + 1 + tid; r < m; r += nt) {
      if (r == k + 1) { v[r] = mkc(1.0, 0.0); H[r + (int64_t)k * m] = mkc(beta, 0.0); }
      else { v[r] = cmul(H[r + (int64_t)k * m], scale); H[r + (int64_t)k * m] = mkc(0.0, 0.0); }
    }
    __syncthreads();
    // left: H[k+1:, j] -= conj(tau) v (v^H H[k+1:, j]),  j > k
    const cplx ctau = cconj(tau);
    for (int j = k + 1 + 2 * warp; j < m; j += 2 * nw) {
      cplx* c0 = H + (int64_t)j * m;
      const bool two = j + 1 < m;
      cplx* c1 = two ? c0 + m : c0;
      cplx d0 = mkc(0.0, 0.0), d1 = mkc(0.0, 0.0);
      for (int r = k + 1 + lane; r < m; r += 32) { const cplx vr = v[r]; cfmac(d0, vr, c0[r]); cfmac(d1, vr, c1[r]); }
      d0 = cmul(ctau, warp_sum(d0)); d1 = cmul(ctau, warp_sum(d1));
      for (int r = k + 1 + lane; r < m; r += 32) {
        const cplx vr = v[r];
        cfms(c0[r], vr, d0);
        if (two) cfms(c1[r], vr, d1);
      }
    }
    __syncthreads();
    // right: H[:, k+1:] -= tau (H[:, k+1:] v) v^H
    constexpr int RS = HESS_THREADS / 2;
    const int sl = tid / RS;   // column slice 0 / 1
    for (int i = tid % RS; i < m; i += RS) {
      cplx a0 = mkc(0.0, 0.0), a1 = mkc(0.0, 0.0);
      int j = k + 1 + sl;
      for (; j + 2 < m; j += 4) { cfma(a0, H[i + (int64_t)j * m], v[j]); cfma(a1, H[i + (int64_t)(j + 2) * m], v[j + 2]); }
      if (j < m) cfma(a0, H[i + (int64_t)j * m], v[j]);
      y[sl * m + i] = cadd(a0, a1);
    }
    __syncthreads();
    for (int i = tid % RS; i < m; i += RS) {
      const cplx acc = cmul(tau, cadd(y[i], y[m + i]));
      for (int j = k + 1 + sl; j < m; j += 2) {
        cplx h = H[i + (int64_t)j * m];
        cfms(h, acc, cconj(v[j]));
        H[i + (int64_t)j * m] = h;
      }
    }
    __syncthreads();
  }
}

// The same reduction with a thread-block CLUSTER per matrix (few Wilson matrices, many idle SMs: 48
// matrices on 148 SMs at the bench workload): the CTAs of a cluster split the columns of the left update
// and the rows of the right update; the reflector is computed redundantly by every CTA, so the only
// communication is the cluster barrier that orders the global-memory updates (3 per column).
__global__ void __launch_bounds__(1024) k_hessenberg_cluster(cplx* __restrict__ W, int m) {
  namespace cg = cooperative_groups;
  cg::cluster_group cluster = cg::this_cluster();
  const int CS = (int)cluster.num_blocks(), rank = (int)cluster.block_rank();
  extern __shared__ cplx vsh[];   // v[m], y[4][rows_per]
  __shared__ double redd[33];
  cplx* v = vsh; cplx* y = vsh + m;
  cplx* H = W + (blockIdx.x / CS) * (int64_t)m * m;
  const int tid = threadIdx.x, nt = 1024, warp = tid >> 5, lane = tid & 31, nw = nt >> 5;
  const int rows_per = (m + CS - 1) / CS;
  const int i0 = rank * rows_per, i1 = (i0 + rows_per < m) ? i0 + rows_per : m;
  for (int k = 0; k < m - 2; ++k) {
    // column k into shared memory (every CTA), norm of its tail
    double ss = 0.0;
    for (int r = k + 1 + tid; r < m; r += nt) {
      const cplx x = H[r + (int64_t)k * m];
      v[r] = x;
      if (r > k + 1) ss += cabs2(x);
    }
    const double xn2 = block_sum(ss, redd);
    const cplx alpha = v[k + 1];
    cluster.sync();                                   // everybody has read column k
    if (xn2 == 0.0 && alpha.y == 0.0) continue;       // (uniform over the cluster)
    const double beta = -copysign(sqrt(cabs2(alpha) + xn2), alpha.x);
    const cplx tau = mkc((beta - alpha.x) / beta, -alpha.y / beta);
    const cplx scale = cdiv(mkc(1.0, 0.0), mkc(alpha.x - beta, alpha.y));
    __syncthreads();                                  // alpha read before v[k+1] is overwritten
    for (int r = k + 1 + tid; r < m; r += nt) {
      const cplx x = v[r];
      v[r] = (r == k + 1) ? mkc(1.0, 0.0) : cmul(x, scale);
      if (rank == 0) H[r + (int64_t)k * m] = (r == k + 1) ? mkc(beta, 0.0) : mkc(0.0, 0.0);
    }
    __syncthreads();
    // left: H[k+1:, j] -= conj(tau) v (v^H H[k+1:, j]),  j > k; column pairs dealt round robin over the cluster
    const cplx ctau = cconj(tau);
    for (int j = k + 1 + 2 * (warp + nw * rank); j < m; j += 2 * nw * CS) {
      cplx* c0 = H + (int64_t)j * m;
      const bool two = j + 1 < m;
      cplx* c1 = two ? c0 + m : c0;
      cplx d0 = mkc(0.0, 0.0), d1 = mkc(0.0, 0.0);
      for (int r = k + 1 + lane; r < m; r += 32) { const cplx vr = v[r]; cfmac(d0, vr, c0[r]); cfmac(d1, vr, c1[r]); }
      d0 = cmul(ctau, warp_sum(d0)); d1 = cmul(ctau, warp_sum(d1));
      for (int r = k + 1 + lane; r < m; r += 32) {
        const cplx vr = v[r];
        cfms(c0[r], vr, d0);
        if (two) cfms(c1[r], vr, d1);
      }
    }
    cluster.sync();                                   // all columns updated before rows are combined
    // right: H[i0:i1, k+1:] -= tau (H[i0:i1, k+1:] v) v^H; thread = (row, column slice of 4)
    const int sl = tid >> 8;
    for (int ib = i0; ib < i1; ib += 256) {
      const int i = ib + (tid & 255);
      if (i < i1) {
        cplx a0 = mkc(0.0, 0.0), a1 = mkc(0.0, 0.0);
        int j = k + 1 + sl;
        for (; j + 4 < m; j += 8) { cfma(a0, H[i + (int64_t)j * m], v[j]); cfma(a1, H[i + (int64_t)(j + 4) * m], v[j + 4]); }
        if (j < m) cfma(a0, H[i + (int64_t)j * m], v[j]);
        y[sl * rows_per + (i - i0)] = cadd(a0, a1);
      }
    }
    __syncthreads();
    for (int ib = i0; ib < i1; ib += 256) {
      const int i = ib + (tid & 255);
      if (i < i1) {
        const int li = i - i0;
        const cplx acc = cmul(tau, cadd(cadd(y[li], y[rows_per + li]), cadd(y[2 * rows_per + li], y[3 * rows_per + li])));
        for (int j = k + 1 + sl; j < m; j += 4) {
          cplx h = H[i + (int64_t)j * m];
          cfms(h, acc, cconj(v[j]));
          H[i + (int64_t)j * m] = h;
        }
      }
    }
    cluster.sync();                                   // rows updated before the next column is read
  }
}

// Givens: c real, s complex with [c s; -conj(s) c] [a; b] = [r; 0]
__device__ __forceinline__ void givens(cplx a, cplx b, double& c, cplx& s) {
  const double nb2 = cabs2(b);
  if (nb2 == 0.0) { c = 1.0; s = mkc(0.0, 0.0); return; }
  const double na2 = cabs2(a);
  if (na2 == 0.0) { c = 0.0; const double nb = sqrt(nb2); s = mkc(b.x / nb, -b.y / nb); return; }
  // the rotation sits on the sequential chain of the sweep: two reciprocal square roots instead of
  // two square roots and three divisions
  const double ia = rsqrt(na2), ir = rsqrt(na2 + nb2);
  c = na2 * ia * ir;                                  // |a| / sqrt(|a|^2 + |b|^2)
  s = cscale(ia * ir, cmulc(b, a));                   // (a / |a|) conj(b) / sqrt(|a|^2 + |b|^2)
}

constexpr int QR_MAXOWN = 4;   // columns / rows owned per thread: m <= 4 * blockDim

// Explicit single-shift QR on the upper Hessenberg matrix H (column-major m x m), eigenvalues only.
__global__ void k_hqr(cplx* __restrict__ W, int m, cplx* __restrict__ lam, int* __restrict__ fail) {
  extern __shared__ double shq[];       // cs[m] (double), sn[m] (cplx)
  double* cs = shq;
  cplx* sn = (cplx*)(shq + ((m + 1) & ~1));
  __shared__ int s_l;
  __shared__ cplx s_sig;
  __shared__ int redi[33];
  cplx* H = W + blockIdx.x * (int64_t)m * m;
  cplx* out = lam + blockIdx.x * (int64_t)m;
  const int tid = threadIdx.x, nt = blockDim.x;
  const int nl = (m + QR_MAXOWN - 1) / QR_MAXOWN <= 64 ? (nt < 64 ? nt : 64) : (nt < 128 ? nt : (m <= QR_MAXOWN * 128 ? 128 : nt));
  const double eps = DBL_EPSILON;
  int hi = m - 1, its = 0, nfail = 0;
  while (hi >= 0) {
    // ---- deflation scan: largest l in (0, hi] with negligible H[l][l-1], else 0
    int best = 0;
    for (int k = hi - tid; k >= 1; k -= nt) {
      const double sub = cabs1(H[k + (int64_t)(k - 1) * m]);
      double sd = cabs1(H[(k - 1) + (int64_t)(k - 1) * m]) + cabs1(H[k + (int64_t)k * m]);
      if (sd == 0.0) sd = 1.0;
      if (sub <= eps * sd) { best = k; break; }   // first hit going down is this thread's largest
    }
    // block max
    for (int o = 16; o > 0; o >>= 1) best = max(best, __shfl_xor_sync(0xffffffffu, best, o));
    __syncthreads();
    if ((tid & 31) == 0) redi[tid >> 5] = best;
    __syncthreads();
    if (tid == 0) {
      int b = 0;
      for (int w = 0; w < (nt + 31) / 32; ++w) b = max(b, redi[w]);
      s_l = b;
      if (b < hi) {
        if (b > 0) H[b + (int64_t)(b - 1) * m] = mkc(0.0, 0.0);
        cplx sig;
        if (its == 10 || its == 20 || its == 30) {
          sig = H[hi + (int64_t)hi * m];
          sig.x += 0.75 * cabs1(H[hi + (int64_t)(hi - 1) * m]);
        } else {
          const cplx a = H[(hi - 1) + (int64_t)(hi - 1) * m], bb = H[(hi - 1) + (int64_t)hi * m];
          const cplx cc = H[hi + (int64_t)(hi - 1) * m], d = H[hi + (int64_t)hi * m];
          cplx l1, l2;
          eig2(a, bb, cc, d, l1, l2);
          sig = (cabs2(csub(l1, d)) <= cabs2(csub(l2, d))) ? l1 : l2;
        }
        s_sig = sig;
      }
    }
    __syncthreads();
    const int l = s_l;
    if (l == hi) {
      if (tid == 0) out[hi] = H[hi + (int64_t)hi * m];
      --hi; its = 0;
      continue;
    }
    ++its;
    if (its > 60) {   // give up on this eigenvalue: take the diagonal entry, flag it
      if (tid == 0) out[hi] = H[hi + (int64_t)hi * m];
      ++nfail; --hi; its = 0;
      continue;
    }
    const cplx sig = s_sig;
    // ---- left phase: R = Q^H (H - sig I).  Thread t < nl owns the QR_MAXOWN CONSECUTIVE columns
    // l + 4t .. l + 4t + 3.  The rotations form a sequential chain (G_s needs column s after G_{s-1});
    // with consecutive columns per thread the owner of a round generates its 4 rotations back to back
    // from registers and publishes them together: one barrier per 4 rotations instead of one per
    // rotation.  Only nl <= 128 threads take part (the barrier spans 4 warps).
    if (tid < nl) {
      const int j0 = l + QR_MAXOWN * tid;
      cplx carry[QR_MAXOWN];
#pragma unroll
      for (int u = 0; u < QR_MAXOWN; ++u) {
        const int j = j0 + u;
        carry[u] = mkc(0.0, 0.0);
        if (j <= hi) { carry[u] = H[l + (int64_t)j * m]; if (j == l) carry[u] = csub(carry[u], sig); }
      }
      const int nrounds = (hi - l + QR_MAXOWN - 1) / QR_MAXOWN;
      for (int r = 0; r < nrounds; ++r) {            // every thread runs every round: the barrier is warp-aligned
        const int sb = l + QR_MAXOWN * r;            // rotations sb .. sb+3 (those < hi)
        // rows sb+1 .. sb+4 of the owned columns (H - sig I); rows ahead of the sweep are not written by it
        cplx Y[QR_MAXOWN][QR_MAXOWN];   // [rotation v][column u]
#pragma unroll
        for (int v = 0; v < QR_MAXOWN; ++v)
#pragma unroll
          for (int u = 0; u < QR_MAXOWN; ++u) {
            const int row = sb + 1 + v, j = j0 + u;
            cplx y = mkc(0.0, 0.0);
            if (r <= tid && row <= hi && j <= hi && j + 1 >= row) { y = H[row + (int64_t)j * m]; if (row == j) y = csub(y, sig); }
            Y[v][u] = y;
          }
        if (r == tid) {
          // owner: generate G_s from the own column s = j0 + v, apply it to the own columns right away
#pragma unroll
          for (int v = 0; v < QR_MAXOWN; ++v) {
            const int sidx = sb + v;
            if (sidx < hi) {
              double c_; cplx s_;
              givens(carry[v], Y[v][v], c_, s_);
              cs[sidx - l] = c_; sn[sidx - l] = s_;
#pragma unroll
              for (int u = 0; u < QR_MAXOWN; ++u)
                if (u >= v && j0 + u <= hi) {
                  const cplx x = carry[u], yv = Y[v][u];
                  cplx top = cscale(c_, x); cfma(top, s_, yv);
                  cplx bot = cscale(c_, yv); cfms(bot, cconj(s_), x);
                  H[sidx + (int64_t)(j0 + u) * m] = top;
                  carry[u] = bot;
                }
            }
          }
        }
        asm volatile("bar.sync 1, %0;" ::"r"(nl) : "memory");   // rotations of round r are published
        if (r < tid) {
#pragma unroll
          for (int v = 0; v < QR_MAXOWN; ++v) {
            const int sidx = sb + v;
            if (sidx < hi) {
              const double c_ = cs[sidx - l];
              const cplx s_ = sn[sidx - l];
#pragma unroll
              for (int u = 0; u < QR_MAXOWN; ++u)
                if (j0 + u <= hi) {
                  const cplx x = carry[u], yv = Y[v][u];
                  cplx top = cscale(c_, x); cfma(top, s_, yv);
                  cplx bot = cscale(c_, yv); cfms(bot, cconj(s_), x);
                  H[sidx + (int64_t)(j0 + u) * m] = top;
                  carry[u] = bot;
                }
            }
          }
        }
      }
#pragma unroll
      for (int u = 0; u < QR_MAXOWN; ++u)
        if (j0 + u == hi) H[hi + (int64_t)hi * m] = carry[u];
    }
    __syncthreads();
    // ---- right phase: H = R Q + sig I; thread owns rows i = l + tid + q*nt, walks along the row
    for (int i = l + tid; i <= hi; i += nt) {
      const int sstart = (i - 1 > l) ? i - 1 : l;
      cplx x = (sstart == i - 1) ? mkc(0.0, 0.0) : H[i + (int64_t)sstart * m];   // R[i][i-1] = 0
      // the row is walked left to right; its elements are prefetched two columns ahead
      cplx y0 = (sstart + 1 <= hi) ? H[i + (int64_t)(sstart + 1) * m] : mkc(0.0, 0.0);
      cplx y1 = (sstart + 2 <= hi) ? H[i + (int64_t)(sstart + 2) * m] : mkc(0.0, 0.0);
      for (int s = sstart; s < hi; ++s) {
        const double c_ = cs[s - l];
        const cplx s_ = sn[s - l];
        const cplx yv = y0;
        y0 = y1;
        if (s + 3 <= hi) y1 = H[i + (int64_t)(s + 3) * m];
        // col s: c x + conj(s) y ; col s+1: -s x + c y
        cplx ns = cscale(c_, x); cfma(ns, cconj(s_), yv);
        cplx n1 = cscale(c_, yv); cfms(n1, s_, x);
        if (s == i) ns = cadd(ns, sig);
        H[i + (int64_t)s * m] = ns;
        x = n1;
      }
      if (i == hi) x = cadd(x, sig);
      H[i + (int64_t)hi * m] = x;
    }
    __syncthreads();
  }
  if (tid == 0 && fail) fail[blockIdx.x] = nfail;
}

// theta = arg(lambda) on (-pi, pi], rank sort ascending (ties by index), |lambda| carried along.
__global__ void k_sort_phases(const cplx* __restrict__ lam, int m, double* __restrict__ theta,
                              double* __restrict__ absl) {
  extern __shared__ double th[];   // m
  const int64_t c = blockIdx.x;
  const cplx* l = lam + c * m;
  for (int i = threadIdx.x; i < m; i += blockDim.x) {
    double t = atan2(l[i].y, l[i].x);
    if (t <= -M_PI) t = M_PI;
    th[i] = t;
  }
  __syncthreads();
  for (int i = threadIdx.x; i < m; i += blockDim.x) {
    const double t = th[i];
    int rank = 0;
    for (int j = 0; j < m; ++j) rank += (th[j] < t) || (th[j] == t && j < i);
    theta[c * m + rank] = t;
    if (absl) absl[c * m + rank] = hypot(l[i].x, l[i].y);
  }
}

}  // namespace

size_t be_eigenphases_scratch_bytes(int64_t cnt, int m) {
  return be_align256((size_t)cnt * m * sizeof(cplx)) + be_align256((size_t)cnt * sizeof(int));
}

int be_eigenvalues_general(be_ctx* ctx, cplx* W, int64_t cnt, int m, cplx* lam, int* fail) {
  cudaStream_t st = ctx->stream;
  if (cnt <= 0) return BE_OK;
  if (m <= 2) {
    k_eig_small<<<(unsigned)((cnt + 127) / 128), 128, 0, st>>>(W, cnt, m, lam);
    ctx->launches++;
    return (int)cudaGetLastError();
  }
  int nt = ((m + 31) / 32) * 32;
  if (nt > 256) nt = (m > QR_MAXOWN * 256) ? 512 : 256;
  if (m > QR_MAXOWN * nt) return BE_ERR_UNSUPPORTED;
  const size_t sh1 = 3 * (size_t)m * sizeof(cplx);
  be_prof_begin(ctx, PK_HESS);
  if (m <= 48) {
    k_hessenberg<64><<<(unsigned)cnt, 64, sh1, st>>>(W, m);
  } else if (m <= 160) {
    k_hessenberg<256><<<(unsigned)cnt, 256, sh1, st>>>(W, m);
  } else {
    // few large matrices: a cluster of CTAs per matrix as long as the clusters fit the machine in one wave
    int cs = 1;
    for (int c = 2; c <= 4; ++c) if (cnt * c <= ctx->sm_count) cs = c;
    if (cs > 1) {
      const size_t shc = ((size_t)m + 4 * (size_t)((m + cs - 1) / cs)) * sizeof(cplx);
      if (shc > 48 * 1024) BE_CUDA(cudaFuncSetAttribute(k_hessenberg_cluster, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)shc));
      cudaLaunchConfig_t cfg = {};
      cfg.gridDim = dim3((unsigned)(cnt * cs)); cfg.blockDim = dim3(1024); cfg.dynamicSmemBytes = shc; cfg.stream = st;
      cudaLaunchAttribute at[1];
      at[0].id = cudaLaunchAttributeClusterDimension;
      at[0].val.clusterDim.x = cs; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
      cfg.attrs = at; cfg.numAttrs = 1;
      if (cudaLaunchKernelEx(&cfg, k_hessenberg_cluster, W, m) != cudaSuccess) { cudaGetLastError(); cs = 1; }   // cluster shape refused
    }
    if (cs == 1) {
      if (sh1 > 48 * 1024) BE_CUDA(cudaFuncSetAttribute(k_hessenberg<1024>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sh1));
      k_hessenberg<1024><<<(unsigned)cnt, 1024, sh1, st>>>(W, m);
    }
  }
  be_prof_end(ctx, PK_HESS, (double)cnt * m * m * 32.0, (double)cnt * (40.0 / 3.0) * m * (double)m * m);
  ctx->launches++;
  BE_CUDA(cudaGetLastError());
  const size_t sh2 = (size_t)((m + 1) & ~1) * sizeof(double) + (size_t)m * sizeof(cplx);
  if (sh2 > 48 * 1024) BE_CUDA(cudaFuncSetAttribute(k_hqr, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sh2));
  be_prof_begin(ctx, PK_HQR);
  k_hqr<<<(unsigned)cnt, nt, sh2, st>>>(W, m, lam, fail);
  be_prof_end(ctx, PK_HQR, (double)cnt * m * m * 32.0, 0.0);
  ctx->launches++;
  return (int)cudaGetLastError();
}

// Numerical trouble must not come back as plausible numbers with rc = 0: the phases of a Wilson matrix whose QR
// iteration gave up (fail), or one of whose eigensolves upstream was flagged (bad: inverse iteration / cluster
// orthogonalization failures, non-finite eigenvalues), are replaced by NaN.
__global__ void k_poison(double* __restrict__ theta, double* __restrict__ absl, const int* __restrict__ fail,
                         const int* __restrict__ bad, int64_t cnt, int m) {
  const int64_t c = blockIdx.x;
  if (!(fail[c] || (bad && bad[c]))) return;
  for (int k = threadIdx.x; k < m; k += blockDim.x) {
    theta[c * m + k] = nan("");
    if (absl) absl[c * m + k] = nan("");
  }
}

int be_eigenphases(be_ctx* ctx, cplx* W, int64_t cnt, int m, double* theta, double* absl, const int* bad) {
  if (cnt <= 0 || m <= 0) return BE_OK;
  cplx* lam = (cplx*)be_arena_alloc(ctx, (size_t)cnt * m * sizeof(cplx));
  int* fail = (int*)be_arena_alloc(ctx, (size_t)cnt * sizeof(int));
  if (!lam || !fail) return BE_ERR_NOMEM;
  BE_CUDA(cudaMemsetAsync(fail, 0, (size_t)cnt * sizeof(int), ctx->stream));
  BE_TRY(be_eigenvalues_general(ctx, W, cnt, m, lam, fail));
  BE_TRY(be_sort_phases(ctx, lam, cnt, m, theta, absl));
  k_poison<<<(unsigned)cnt, 64, 0, ctx->stream>>>(theta, absl, fail, bad, cnt, m);
  ctx->launches++;
  return (int)cudaGetLastError();
}

int be_sort_phases(be_ctx* ctx, const cplx* lam, int64_t cnt, int m, double* theta, double* absl) {
  int nt = ((m + 31) / 32) * 32;
  if (nt > 256) nt = 256;
  const size_t sh = (size_t)m * sizeof(double);
  if (sh > 48 * 1024) BE_CUDA(cudaFuncSetAttribute(k_sort_phases, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sh));
  k_sort_phases<<<(unsigned)cnt, nt, sh, ctx->stream>>>(lam, m, theta, absl);
  ctx->launches++;
  return (int)cudaGetLastError();
}
