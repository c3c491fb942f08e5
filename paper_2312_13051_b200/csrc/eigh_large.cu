// S1 -- batched complex128 Hermitian eigensolver for N > 8 ("exact diagonalization
// of a discretized Hamiltonian at many points in reciprocal space" is where the time goes).
//
// All matrices of a chunk advance in lock step, one kernel launch per algorithmic step over the
// whole batch, so every launch is a wide streaming kernel:
//   S1a  blocked Householder tridiagonalization  B = Q T Q^H  (panel width NB = 32)
//          k_colw  : finish w_i (panel corrections, tau, -1/2 tau (w^H v) v) and, in the same sweep
//                    over the panels, apply the pending updates to column i+1 and generate its reflector
//          k_hemv  : y = B22 v on the lower triangle only (each element read once, used twice)
//          rank-2k : B22 -= V W^H + W V^H                   -> DMMA ZGEMM (zgemm.cu), lower tiles
//   S1b  real symmetric tridiagonal eigenproblem
//          k_bisect: all eigenvalues by Sturm-count bisection, one thread per eigenvalue
//          k_invit : inverse iteration, one thread per eigenvector (pivoted LU of T - lambda I)
//          cluster_orth.cu: orthogonalization inside clusters of close eigenvalues (CGS2 for small
//                    clusters, Cholesky-QR on DMMA for big ones), then one refinement solve
//   S1c  compact-WY back-transform  U = conj(Q) Z            -> DMMA ZGEMMs
//
// Memory view: the row-major Hermitian input H, read as a column-major array, is B = conj(H).
// B is reduced on its lower triangle; eigenvectors of H are the conjugates of those of B, which
// is obtained for free by back-transforming with conjugated reflectors (Z is real).
#include "be_common.cuh"
#include "tma.cuh"
#include <float.h>

namespace {

constexpr int NB = 32;    // panel width of the tridiagonalization
constexpr int NBT = 128;  // width of the compact-WY blocks of the back-transform (4 panels)
constexpr int HB = 32;    // block-column width of the symmetric matrix-vector kernel
constexpr double SPLIT_TOL = 32.0;     // |e_i| <= max(SPLIT_TOL, N) * eps * ||T|| splits the tridiagonal matrix
                                       // (the backward error of the reduction itself is O(N eps ||T||))
constexpr double CLUSTER_TOL = 2e-5;   // eigenvalues closer than this (relative to ||T||) are re-orthogonalized:
                                       // inverse-iteration vectors of eigenvalues a gap g apart are orthogonal to
                                       // ~eps ||T|| / g, i.e. <= 1e-11 outside clusters (LAPACK's 1e-3 buys eps-level
                                       // orthogonality the 1e-8 phase tolerance does not need, at the price of
                                       // clusters of 50-90 vectors on the N = 1600 supercell)

// ------------------------------------------------------------------------------------------
__global__ void k_gather(const cplx* __restrict__ H, cplx* __restrict__ Bw, GridMap map,
                         int64_t loop0, int N, int nchunk) {
  const int64_t c = blockIdx.x / nchunk;
  const int part = blockIdx.x % nchunk;
  const int64_t src = gridmap_index(map, loop0 + c / map.n1, (int)(c % map.n1));
  const cplx* s = H + src * (int64_t)N * N;
  cplx* d = Bw + c * (int64_t)N * N;
  const int64_t nn = (int64_t)N * N;
  for (int64_t idx = (int64_t)part * 2048 + threadIdx.x; idx < nn && idx < (int64_t)(part + 1) * 2048; idx += blockDim.x)
    d[idx] = s[idx];
}

// ------------------------------------------------------------------------------------------
// y = B22 v with B22 = B[i+1:, i+1:] Hermitian, lower triangle stored; v = B[i+1:, i].
//
// The kernel is HBM bound (1 flop/byte): every element B[r][c], r > c, is read exactly once and used
// twice, for y[r] (row part) and for y[c] (column part).  CTA = (matrix, block column J of HB = 32
// columns).  A producer warp streams the block column through shared memory in stages of
// HROWS = 64 rows with TMA bulk copies (cp.async.bulk, one per column segment plus one for the
// matching piece of v, completion on an mbarrier), HSTAGES deep, so the bytes in flight do not
// depend on registers or on the progress of the arithmetic.  256 consumer threads: thread =
// (row lr of the stage, group cg of 8 columns).  Row part: summed over the 4 column groups through
// shared memory and written per block column to P (k_colw adds the block columns up: no atomics, the
// result is bitwise reproducible).  Column part: 8 accumulators per thread kept in registers over
// the whole block column, reduced once at the end and written to zpart.
constexpr int HROWS = 64;
constexpr int HSTAGES = 3;
constexpr int HEMV_THREADS = 256 + 32;
constexpr int HSTAGE_ELEMS = (HB + 1) * HROWS;                 // 32 columns + the v segment
constexpr size_t HEMV_SMEM = (size_t)HSTAGES * HSTAGE_ELEMS * sizeof(cplx) + 2 * 4 * HROWS * sizeof(cplx)
                             + 2 * HSTAGES * sizeof(unsigned long long) + 8 * sizeof(int) + 64 + 2 * 64 * sizeof(cplx);

// The kernel is PERSISTENT: 2 CTAs per SM fetch work items (matrix, block column) from a global
// counter until none is left (panel blocks and long block columns come first in the item order).
// The producer warp runs ahead of the consumers across item boundaries -- the stage counter never
// restarts -- so the prologue / epilogue of one item is covered by the stream of the next and a
// single resident CTA keeps its share of HBM busy (which is what lets the FP64-bound GEMMs of the
// previous chunk share the SM in the chunk pipeline).  Item numbers travel from the producer to the
// consumers through a small ring in shared memory, ordered by the stages' mbarriers.
constexpr int HRING = 8;
__global__ void __launch_bounds__(HEMV_THREADS, 2) k_hemv(const cplx* __restrict__ Bw, cplx* __restrict__ P,
                                                          cplx* __restrict__ zpart, int N, int i, int nJ, int nJmax,
                                                          const cplx* __restrict__ Wp, cplx* __restrict__ pqg,
                                                          int p, int npb, int* __restrict__ counter, int total) {
  extern __shared__ __align__(128) unsigned char hsm[];
  cplx* stage = (cplx*)hsm;                                           // [HSTAGES][HB + 1][HROWS]
  cplx* ysm = stage + (size_t)HSTAGES * HSTAGE_ELEMS;                 // [2][4][HROWS]
  unsigned long long* full = (unsigned long long*)(ysm + 2 * 4 * HROWS);
  unsigned long long* empty = full + HSTAGES;
  volatile int* ring = (volatile int*)(empty + HSTAGES);              // [HRING] item numbers, -1 = end
  cplx* zsm0 = (cplx*)(hsm + HEMV_SMEM - 2 * 64 * sizeof(cplx));      // [2][8 warps][8]
  const int per = nJ + npb;                                           // items per matrix
  const int k = i - p;
  const int tid = threadIdx.x;
  if (tid == 0) {
    for (int s = 0; s < HSTAGES; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 8); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  if (tid >= 256) {
    // ---- producer warp: lane = column of the block column (lane 0 also copies the v segment)
    const int lane = tid - 256;
    int gs = 0;
    int next = 0;
    if (lane == 0) next = atomicAdd(counter, 1);
    for (int seq = 0;; ++seq) {
      // the item after this one is fetched now: the atomic's round trip hides behind the copies
      const int item = __shfl_sync(0xffffffffu, next, 0);
      if (lane == 0 && item < total) next = atomicAdd(counter, 1);
      if (item >= total) {
        // end of work: one empty stage carries the stop mark
        const int slot = gs % HSTAGES;
        if (gs >= HSTAGES) mbar_wait(&empty[slot], ((gs / HSTAGES) - 1) & 1);
        if (lane == 0) { ring[seq % HRING] = -1; mbar_arrive(&full[slot]); }
        break;
      }
      const int64_t c = item / per;
      const int u = item % per;
      const bool panel = u < npb;
      const int J = panel ? u : u - npb;
      const cplx* __restrict__ B = Bw + c * (int64_t)N * N;
      const cplx* __restrict__ W = Wp + c * (int64_t)N * NB;
      const cplx* __restrict__ v = B + (int64_t)i * N;
      const int q0 = panel ? J * HB : 0;
      const int c0 = panel ? i + 1 : i + 1 + J * HB;
      const int ncols = panel ? ((2 * k - q0 < HB) ? 2 * k - q0 : HB) : ((N - c0 < HB) ? N - c0 : HB);
      const int nst = (N - c0 + HROWS - 1) / HROWS;
      const cplx* src = nullptr;
      if (lane < ncols) {
        const int q = q0 + lane;
        src = !panel ? B + (int64_t)(c0 + lane) * N : (q < k ? W + (int64_t)q * N : B + (int64_t)(p + q - k) * N);
      }
      for (int s = 0; s < nst; ++s, ++gs) {
        const int slot = gs % HSTAGES;
        if (gs >= HSTAGES) mbar_wait(&empty[slot], ((gs / HSTAGES) - 1) & 1);
        const int r0 = c0 + s * HROWS;
        const int nr = (N - r0 < HROWS) ? N - r0 : HROWS;
        const uint32_t seg = (uint32_t)nr * sizeof(cplx);
        cplx* dst = stage + (size_t)slot * HSTAGE_ELEMS;
        if (lane == 0) {
          if (s == 0) ring[seq % HRING] = item;      // published by the release of the arrive below
          mbar_expect_tx(&full[slot], seg * (uint32_t)(ncols + 1));
          tma_bulk_g2s(dst + HB * HROWS, v + r0, seg, &full[slot]);
        }
        __syncwarp();
        if (src) tma_bulk_g2s(dst + lane * HROWS, src + r0, seg, &full[slot]);
      }
    }
    return;
  }

  // ---- consumers
  const int lr = tid & (HROWS - 1), cg = tid >> 6, lane = tid & 31, warp = tid >> 5;
  int gs = 0;
  for (int seq = 0;; ++seq) {
    mbar_wait(&full[gs % HSTAGES], (gs / HSTAGES) & 1);   // first stage of the item (or the stop mark)
    const int item = ring[seq % HRING];
    if (item < 0) break;
    const int64_t c = item / per;
    const int u = item % per;
    const bool panel = u < npb;
    const int J = panel ? u : u - npb;
    const int q0 = panel ? J * HB : 0;
    const int c0 = panel ? i + 1 : i + 1 + J * HB;
    const int ncols = panel ? ((2 * k - q0 < HB) ? 2 * k - q0 : HB) : ((N - c0 < HB) ? N - c0 : HB);
    const int nst = (N - c0 + HROWS - 1) / HROWS;
    int nq = ncols - cg * 8;
    nq = nq < 0 ? 0 : (nq > 8 ? 8 : nq);
    cplx vc[8], accz[8];
    {
      // v at the block column's own columns = the head of the first stage's v segment (rows c0 ..)
      const cplx* v0 = stage + (size_t)(gs % HSTAGES) * HSTAGE_ELEMS + HB * HROWS;
#pragma unroll
      for (int q = 0; q < 8; ++q) {
        accz[q] = mkc(0.0, 0.0);
        vc[q] = (q < nq && !panel) ? v0[cg * 8 + q] : mkc(0.0, 0.0);
      }
    }
    cplx* Prow = P + (c * nJmax + J) * (int64_t)N;
    for (int s = 0; s < nst; ++s, ++gs) {
      const int slot = gs % HSTAGES;
      const cplx* st = stage + (size_t)slot * HSTAGE_ELEMS;
      const int r = c0 + s * HROWS + lr;
      if (s > 0) mbar_wait(&full[slot], (gs / HSTAGES) & 1);
      cplx yr = mkc(0.0, 0.0);
      if (r < N) {
        const cplx vr = st[HB * HROWS + lr];
        if (panel) {
#pragma unroll
          for (int q = 0; q < 8; ++q)
            if (q < nq) cfmac(accz[q], st[(cg * 8 + q) * HROWS + lr], vr);
        } else if (s > 0) {
          if (nq == 8) {
            cplx a[8];
#pragma unroll
            for (int q = 0; q < 8; ++q) a[q] = st[(cg * 8 + q) * HROWS + lr];
#pragma unroll
            for (int q = 0; q < 8; ++q) { cfma(yr, a[q], vc[q]); cfmac(accz[q], a[q], vr); }
          } else {
#pragma unroll
            for (int q = 0; q < 8; ++q)
              if (q < nq) { const cplx a = st[(cg * 8 + q) * HROWS + lr]; cfma(yr, a, vc[q]); cfmac(accz[q], a, vr); }
          }
        } else {
          // first stage: holds the diagonal block (upper triangle is not part of the matrix)
#pragma unroll
          for (int q = 0; q < 8; ++q)
            if (q < nq) {
              const int col = c0 + cg * 8 + q;
              const cplx a = st[(cg * 8 + q) * HROWS + lr];
              if (r > col) { cfma(yr, a, vc[q]); cfmac(accz[q], a, vr); }
              else if (r == col) { yr.x = fma(a.x, vc[q].x, yr.x); yr.y = fma(a.x, vc[q].y, yr.y); }
            }
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(&empty[slot]);          // this warp is done with the stage
      if (panel) continue;                               // no row part
      cplx* yb = ysm + (gs & 1) * 4 * HROWS;
      yb[cg * HROWS + lr] = yr;
      asm volatile("bar.sync 1, 256;" ::: "memory");     // consumers only
      if (tid < HROWS && r < N) {
        cplx t = cadd(cadd(yb[tid], yb[HROWS + tid]), cadd(yb[2 * HROWS + tid], yb[3 * HROWS + tid]));
        Prow[r] = t;
      }
    }
    // column part: reduce over the 64 rows (2 warps per column group); zsm is double buffered by item
    cplx* zsm = zsm0 + (seq & 1) * 64;   // [8 warps][8]
    {
      // 8 sums over the 32 lanes with 9 exchanges per component (halving the live values at every
      // step) instead of 8 x 5: lane bits 4, 3, 2 end up selecting which of the 8 sums the lane holds
      cplx b4[4], b2[2], b1;
      const bool u16 = lane & 16, u8 = lane & 8, u4 = lane & 4;
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const cplx snd = u16 ? accz[j] : accz[j + 4], kp = u16 ? accz[j + 4] : accz[j];
        b4[j] = mkc(kp.x + __shfl_xor_sync(0xffffffffu, snd.x, 16), kp.y + __shfl_xor_sync(0xffffffffu, snd.y, 16));
      }
#pragma unroll
      for (int j = 0; j < 2; ++j) {
        const cplx snd = u8 ? b4[j] : b4[j + 2], kp = u8 ? b4[j + 2] : b4[j];
        b2[j] = mkc(kp.x + __shfl_xor_sync(0xffffffffu, snd.x, 8), kp.y + __shfl_xor_sync(0xffffffffu, snd.y, 8));
      }
      {
        const cplx snd = u4 ? b2[0] : b2[1], kp = u4 ? b2[1] : b2[0];
        b1 = mkc(kp.x + __shfl_xor_sync(0xffffffffu, snd.x, 4), kp.y + __shfl_xor_sync(0xffffffffu, snd.y, 4));
      }
      b1.x += __shfl_xor_sync(0xffffffffu, b1.x, 2); b1.y += __shfl_xor_sync(0xffffffffu, b1.y, 2);
      b1.x += __shfl_xor_sync(0xffffffffu, b1.x, 1); b1.y += __shfl_xor_sync(0xffffffffu, b1.y, 1);
      if ((lane & 3) == 0) zsm[warp * 8 + (u16 ? 4 : 0) + (u8 ? 2 : 0) + (u4 ? 1 : 0)] = b1;
    }
    asm volatile("bar.sync 1, 256;" ::: "memory");
    if (tid < HB && tid < ncols) {
      const int g = tid >> 3, q = tid & 7;
      const cplx z = cadd(zsm[(2 * g) * 8 + q], zsm[(2 * g + 1) * 8 + q]);
      if (panel) pqg[c * (2 * NB) + q0 + tid] = z;
      else zpart[c * N + c0 + tid] = z;
    }
  }
}

// ------------------------------------------------------------------------------------------
// Fused panel step, one CTA per matrix.
//   do_w  : finish w_i = tau (y - V (W^H v) - W (V^H v)), w_i += -1/2 tau (w_i^H v) v, stored as column
//           k = i - p of the W panel.  y = zpart + sum_J P[J] (k_hemv), the 2k dot products W^H v,
//           V^H v come from the dot CTAs of the same k_hemv launch (pqg).
//   do_col: column ic (= i + 1 with do_w, = i without) gets the pending panel updates
//           B[ic:, ic] -= V[ic:, :kc] conj(W[ic, :kc]) + W[ic:, :kc] conj(V[ic, :kc]) and its reflector
//           is generated (zlarfg): d[ic], e[ic], tau[ic], v stored in place with a unit head.
// With both flags the V and W panels are read ONCE: the column update of ic is accumulated in the
// same sweep that corrects y, the term of the new reflector i is added from shared memory.
constexpr int CW_THREADS = 192;   // 5 CTAs per SM: a chunk of 600 matrices is resident in one wave on 148 SMs (320 threads, 3 per SM: two rounds, 38.6 ms)
__global__ void __launch_bounds__(CW_THREADS, 5) k_colw(cplx* __restrict__ Bw, cplx* __restrict__ Wp,
                                                     const cplx* __restrict__ P, const cplx* __restrict__ zpart,
                                                     const cplx* __restrict__ pqg, double* __restrict__ dd,
                                                     double* __restrict__ ee, cplx* __restrict__ tau,
                                                     int N, int i, int p, int nJmax, int do_w, int do_col) {
  extern __shared__ cplx ysh[];   // w[N] (indexed by global row), then a2[N]
  __shared__ cplx pq[2 * NB], cw2[NB], cv2[NB];
  __shared__ cplx redc[33];
  __shared__ double redd[33];
  __shared__ cplx sh_alpha;
  cplx* a2s = ysh + N;
  const int64_t c = blockIdx.x;
  cplx* __restrict__ B = Bw + c * (int64_t)N * N;
  cplx* __restrict__ W = Wp + c * (int64_t)N * NB;
  const int tid = threadIdx.x;
  const int ic = do_w ? i + 1 : i;
  if (do_w) {
    const cplx* __restrict__ v = B + (int64_t)i * N;
    const int k = i - p;
    if (tid < 2 * k) pq[tid] = pqg[c * (2 * NB) + tid];
    if (do_col && tid < k) {
      cw2[tid] = cconj(W[ic + (int64_t)tid * N]);
      cv2[tid] = cconj(B[ic + (int64_t)(p + tid) * N]);
    }
    __syncthreads();
    const cplx t = tau[c * N + i];
    cplx dot = mkc(0.0, 0.0);
    for (int r = i + 1 + tid; r < N; r += CW_THREADS) {
      cplx y = zpart[c * N + r];
      const int Jr = (r - (i + 1)) / HB;
      cplx a2 = do_col ? B[r + (int64_t)ic * N] : mkc(0.0, 0.0);
      {
        const cplx* Pr = P + c * nJmax * (int64_t)N + r;
        int J = 0;
        for (; J + 4 <= Jr + 1; J += 4) {   // independent loads first: the sweep is latency bound
          const cplx p0 = Pr[(int64_t)J * N], p1 = Pr[(int64_t)(J + 1) * N], p2 = Pr[(int64_t)(J + 2) * N],
                     p3 = Pr[(int64_t)(J + 3) * N];
          y = cadd(cadd(y, cadd(p0, p1)), cadd(p2, p3));
        }
        for (; J <= Jr; ++J) y = cadd(y, Pr[(int64_t)J * N]);
      }
      int cc = 0;
      for (; cc + 4 <= k; cc += 4) {
        cplx bv[4], wv[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) { bv[u] = B[r + (int64_t)(p + cc + u) * N]; wv[u] = W[r + (int64_t)(cc + u) * N]; }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          cfms(y, bv[u], pq[cc + u]);
          cfms(y, wv[u], pq[k + cc + u]);
          if (do_col) { cfms(a2, bv[u], cw2[cc + u]); cfms(a2, wv[u], cv2[cc + u]); }
        }
      }
      for (; cc < k; ++cc) {
        const cplx bv = B[r + (int64_t)(p + cc) * N], wv = W[r + (int64_t)cc * N];
        cfms(y, bv, pq[cc]);
        cfms(y, wv, pq[k + cc]);
        if (do_col) { cfms(a2, bv, cw2[cc]); cfms(a2, wv, cv2[cc]); }
      }
      const cplx wv = cmul(t, y);
      ysh[r] = wv;
      a2s[r] = a2;
      cfmac(dot, wv, v[r]);
    }
    dot = block_sum(dot, redc);
    const cplx al = cmul(mkc(-0.5 * t.x, -0.5 * t.y), dot);
    for (int r = i + 1 + tid; r < N; r += CW_THREADS) {
      cplx wv = ysh[r];
      cfma(wv, al, v[r]);
      W[r + (int64_t)k * N] = wv;
      ysh[r] = wv;
    }
    __syncthreads();
    if (!do_col) return;
    // term of reflector i itself: V[r][k] = v[r] (v[ic] = 1), W[r][k] = w[r]
    const cplx cwi = cconj(ysh[ic]);
    for (int r = ic + tid; r < N; r += CW_THREADS) {
      cplx a2 = a2s[r];
      cfms(a2, v[r], cwi);
      a2 = csub(a2, ysh[r]);
      a2s[r] = a2;
    }
  } else {
    for (int r = ic + tid; r < N; r += CW_THREADS) a2s[r] = B[r + (int64_t)ic * N];
  }
  // ---- zlarfg on column ic (each thread re-reads only the rows it wrote)
  double ss = 0.0;
  for (int r = ic + tid; r < N; r += CW_THREADS) {
    const cplx a2 = a2s[r];
    if (r == ic) dd[c * N + ic] = a2.x;
    else if (r == ic + 1) sh_alpha = a2;
    else ss += cabs2(a2);
  }
  if (ic >= N - 1) return;
  const double xn2 = block_sum(ss, redd);
  const cplx alpha = sh_alpha;
  double beta; cplx t, scale;
  if (xn2 == 0.0 && alpha.y == 0.0) {
    beta = alpha.x; t = mkc(0.0, 0.0); scale = mkc(0.0, 0.0);
  } else {
    beta = -copysign(sqrt(cabs2(alpha) + xn2), alpha.x);
    t = mkc((beta - alpha.x) / beta, -alpha.y / beta);
    scale = cdiv(mkc(1.0, 0.0), mkc(alpha.x - beta, alpha.y));
  }
  for (int r = ic + tid; r < N; r += CW_THREADS) {
    cplx a2 = a2s[r];
    if (r == ic) a2.y = 0.0;
    else if (r == ic + 1) a2 = mkc(1.0, 0.0);
    else a2 = cmul(a2, scale);
    B[r + (int64_t)ic * N] = a2;
  }
  if (tid == 0) { ee[c * N + ic] = beta; tau[c * N + ic] = t; }
}

// ------------------------------------------------------------------------------------------
// Sturm-count bisection: one thread per eigenvalue index, d and e^2 in shared memory.
__global__ void __launch_bounds__(128) k_bisect(const double* __restrict__ dd, const double* __restrict__ ee,
                                                double* __restrict__ lam, double* __restrict__ tnorm,
                                                double* __restrict__ blo, double* __restrict__ bhi,
                                                int* __restrict__ bcl, int N, int nblk, int ne) {
  extern __shared__ double sh[];   // d[N], e2[N]
  __shared__ double rmin[4], rmax[4], remax[4];
  double* d = sh; double* e2 = sh + N;
  const int64_t c = blockIdx.x / nblk;
  const int kb = blockIdx.x % nblk;
  const int tid = threadIdx.x;
  double lmin = DBL_MAX, lmax = -DBL_MAX, emax = 0.0;
  for (int r = tid; r < N; r += 128) {
    const double di = dd[c * N + r];
    const double el = (r > 0) ? fabs(ee[c * N + r - 1]) : 0.0;
    const double er = (r < N - 1) ? fabs(ee[c * N + r]) : 0.0;
    d[r] = di; e2[r] = er * er;
    lmin = fmin(lmin, di - el - er); lmax = fmax(lmax, di + el + er); emax = fmax(emax, er * er);
  }
  for (int o = 16; o > 0; o >>= 1) {
    lmin = fmin(lmin, __shfl_xor_sync(0xffffffffu, lmin, o));
    lmax = fmax(lmax, __shfl_xor_sync(0xffffffffu, lmax, o));
    emax = fmax(emax, __shfl_xor_sync(0xffffffffu, emax, o));
  }
  if ((tid & 31) == 0) { rmin[tid >> 5] = lmin; rmax[tid >> 5] = lmax; remax[tid >> 5] = emax; }
  __syncthreads();
  double gl = fmin(fmin(rmin[0], rmin[1]), fmin(rmin[2], rmin[3]));
  double gu = fmax(fmax(rmax[0], rmax[1]), fmax(rmax[2], rmax[3]));
  emax = fmax(fmax(remax[0], remax[1]), fmax(remax[2], remax[3]));
  const double eps = DBL_EPSILON;
  double tn = fmax(fabs(gl), fabs(gu));
  if (tn == 0.0) tn = DBL_MIN;
  gl -= 2.0 * tn * eps * N + 2.0 * DBL_MIN;
  gu += 2.0 * tn * eps * N + 2.0 * DBL_MIN;
  const double pivmin = DBL_MIN * fmax(1.0, tn * tn);
  (void)emax;
  const int k = kb * 128 + tid;
  if (kb == 0 && tid == 0) tnorm[c] = tn;
  // negligible couplings are dropped (T splits into unreduced blocks); k_invit applies the same rule
  const double split = fmax(SPLIT_TOL, (double)N) * DBL_EPSILON * tn;
  for (int r = tid; r < N; r += 128) if (e2[r] <= split * split) e2[r] = 0.0;
  __syncthreads();
  if (k >= ne) return;   // only the ne lowest eigenvalues are wanted
  double lo = gl, hi = gu;
  int cnt_lo = 0;
  const double atol = 0.25 * eps * tn;
  // A fixed depth for every eigenvalue of the matrix: all final intervals are cells of one dyadic
  // grid, so eigenvalues that cannot be separated share the same cell and k_invit can assign them
  // to blocks consistently.
  int depth = (int)ceil(log2((gu - gl) / atol)) + 1;
  depth = depth < 1 ? 1 : (depth > 120 ? 120 : depth);
  for (int it = 0; it < depth; ++it) {
    const double mid = 0.5 * (lo + hi);
    if (!(mid > lo && mid < hi)) break;
    int cnt = 0;
    double q = d[0] - mid;
    if (fabs(q) < pivmin) q = -pivmin;
    cnt += (q < 0.0);
    for (int r = 1; r < N; ++r) {
      q = d[r] - mid - e2[r - 1] * __drcp_rn(q);   // same expression in k_invit's block search (counts must agree)
      if (fabs(q) < pivmin) q = -pivmin;
      cnt += (q < 0.0);
    }
    if (cnt > k) hi = mid; else { lo = mid; cnt_lo = cnt; }
  }
  lam[c * N + k] = 0.5 * (lo + hi);
  blo[c * N + k] = lo; bhi[c * N + k] = hi; bcl[c * N + k] = cnt_lo;
}

// The same bisection for few wanted eigenvalues (ne <= 64): a block serves mpb = 128 / ne matrices, so
// that the warps are full (config 5: ne = 33 left one lane alone in the second warp of every block).
// Same arithmetic as k_bisect in every step (min / max reductions are exact), hence the same bits.
__global__ void __launch_bounds__(128) k_bisect_packed(const double* __restrict__ dd, const double* __restrict__ ee,
                                                       double* __restrict__ lam, double* __restrict__ tnorm,
                                                       double* __restrict__ blo, double* __restrict__ bhi,
                                                       int* __restrict__ bcl, int N, int64_t count, int ne, int mpb) {
  extern __shared__ double sh[];   // per matrix of the block: d[N], |e|[N], e2[N]
  const int tid = threadIdx.x;
  const int64_t c0 = (int64_t)blockIdx.x * mpb;
  for (int idx = tid; idx < mpb * N; idx += 128) {
    const int mi = idx / N, r = idx % N;
    const int64_t c = c0 + mi;
    double di = 0.0, er = 0.0;
    if (c < count) { di = dd[c * N + r]; er = (r < N - 1) ? fabs(ee[c * N + r]) : 0.0; }
    sh[mi * 3 * N + r] = di; sh[mi * 3 * N + N + r] = er;
  }
  __syncthreads();
  const int mi = tid / ne, k = tid % ne;
  const int64_t c = c0 + mi;
  const bool live = mi < mpb && c < count;
  const double* d = sh + (live ? mi : 0) * 3 * N;
  const double* ea = d + N;
  double* e2 = sh + (live ? mi : 0) * 3 * N + 2 * N;
  double gl = DBL_MAX, gu = -DBL_MAX;
  for (int r = 0; r < N; ++r) {
    const double el = (r > 0) ? ea[r - 1] : 0.0, er = ea[r];
    gl = fmin(gl, d[r] - el - er); gu = fmax(gu, d[r] + el + er);
  }
  const double eps = DBL_EPSILON;
  double tn = fmax(fabs(gl), fabs(gu));
  if (tn == 0.0) tn = DBL_MIN;
  gl -= 2.0 * tn * eps * N + 2.0 * DBL_MIN;
  gu += 2.0 * tn * eps * N + 2.0 * DBL_MIN;
  const double pivmin = DBL_MIN * fmax(1.0, tn * tn);
  const double split = fmax(SPLIT_TOL, (double)N) * DBL_EPSILON * tn;
  if (live) {
    if (k == 0) tnorm[c] = tn;
    for (int r = k; r < N; r += ne) { const double v = ea[r] * ea[r]; e2[r] = (v <= split * split) ? 0.0 : v; }
  }
  __syncthreads();
  if (!live) return;
  double lo = gl, hi = gu;
  int cnt_lo = 0;
  const double atol = 0.25 * eps * tn;
  int depth = (int)ceil(log2((gu - gl) / atol)) + 1;
  depth = depth < 1 ? 1 : (depth > 120 ? 120 : depth);
  for (int it = 0; it < depth; ++it) {
    const double mid = 0.5 * (lo + hi);
    if (!(mid > lo && mid < hi)) break;
    int cnt = 0;
    double q = d[0] - mid;
    if (fabs(q) < pivmin) q = -pivmin;
    cnt += (q < 0.0);
    for (int r = 1; r < N; ++r) {
      q = d[r] - mid - e2[r - 1] * __drcp_rn(q);
      if (fabs(q) < pivmin) q = -pivmin;
      cnt += (q < 0.0);
    }
    if (cnt > k) hi = mid; else { lo = mid; cnt_lo = cnt; }
  }
  lam[c * N + k] = 0.5 * (lo + hi);
  blo[c * N + k] = lo; bhi[c * N + k] = hi; bcl[c * N + k] = cnt_lo;
}

// ------------------------------------------------------------------------------------------
// Inverse iteration, one thread per (matrix, vector).  Pivoted LU of T - sigma I (row
// interchanges between neighbours only), factors kept in global memory laid out [row][vector] so
// that the threads of a warp touch consecutive addresses.
__device__ __forceinline__ double hash_uniform(uint64_t x) {
  x += 0x9E3779B97F4A7C15ull; x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull;
  x = (x ^ (x >> 27)) * 0x94D049BB133111EBull; x ^= x >> 31;
  return (double)(x >> 11) * (2.0 / 9007199254740992.0) - 1.0;
}

__global__ void __launch_bounds__(128) k_invit(const double* __restrict__ dd, const double* __restrict__ ee,
                                               const double* __restrict__ lam, const double* __restrict__ tnorm,
                                               double* __restrict__ fa, double* __restrict__ fb,
                                               double* __restrict__ fc, unsigned char* __restrict__ fp,
                                               int* __restrict__ blk, const double* __restrict__ blo,
                                               const double* __restrict__ bhi, const int* __restrict__ bcl,
                                               double* __restrict__ Z, int N, int nv,
                                               int nvb, int refine, int iters) {
  extern __shared__ double sh[];   // d[N], e[N]
  double* d = sh; double* e = sh + N;
  const int64_t c = blockIdx.x / nvb;
  const int vb = blockIdx.x % nvb;
  const double tn = tnorm[c];
  // pivot floor; the absolute part keeps the squared norm of a solve finite for a matrix that is exactly zero
  const double tol = fmax(DBL_EPSILON * tn, 1e-145);
  // T is split where an off-diagonal entry is negligible: eigenvectors live on one unreduced block,
  // which makes vectors of exactly degenerate eigenvalues (different blocks) orthogonal for free.
  for (int r = threadIdx.x; r < N; r += 128) {
    d[r] = dd[c * N + r];
    double er = (r < N - 1) ? ee[c * N + r] : 0.0;
    { const double sp = fmax(SPLIT_TOL, (double)N) * DBL_EPSILON * tn; if (er * er <= sp * sp) er = 0.0; }   // as in k_bisect
    e[r] = er;
  }
  __syncthreads();
  const int v = vb * 128 + threadIdx.x;
  if (v >= nv) return;
  const double* l = lam + c * N;
  const double sig = l[v];
  const int64_t base = c * (int64_t)N * nv + v;   // element (row r) at base + r*nv
  int bs = 0, be = N - 1;
  if (!refine) {
    // Which unreduced block owns the v-th eigenvalue: bisection ended with count(lo) <= v <
    // count(hi); the Sturm count of the split matrix is the sum of the block counts (same
    // arithmetic as k_bisect), so walking the blocks in order and counting their eigenvalues in
    // (lo, hi] locates instance number v - count(lo) exactly.
    const double xm = blo[c * N + v], xp = bhi[c * N + v];
    int rem = v - bcl[c * N + v];
    const double pivmin = DBL_MIN * fmax(1.0, tn * tn);
    int cm = 0, cp = 0, start = 0;
    bool found = false;
    double qm = 0.0, qp = 0.0;
    for (int r = 0; r < N; ++r) {
      if (r == start) { qm = d[r] - xm; qp = d[r] - xp; }
      else { const double e2 = e[r - 1] * e[r - 1]; qm = d[r] - xm - e2 * __drcp_rn(qm); qp = d[r] - xp - e2 * __drcp_rn(qp); }
      if (fabs(qm) < pivmin) qm = -pivmin;
      if (fabs(qp) < pivmin) qp = -pivmin;
      cm += (qm < 0.0); cp += (qp < 0.0);
      if (r == N - 1 || e[r] == 0.0) {   // end of a block
        const int inst = cp - cm;
        if (rem >= 0 && rem < inst) { bs = start; be = r; found = true; break; }
        rem -= inst;
        cm = 0; cp = 0; start = r + 1;
      }
    }
    if (!found) { bs = 0; be = N - 1; }
    // when the fallback spans several blocks the zero couplings are harmless for the pivoted LU
    blk[(c * nv + v) * 2] = bs; blk[(c * nv + v) * 2 + 1] = be;
    double ai = d[bs] - sig, bi = e[bs];
    for (int r = bs; r < be; ++r) {
      const double sub = e[r];
      const double nd = d[r + 1] - sig;
      const double ns = (r + 1 < be) ? e[r + 1] : 0.0;
      const bool swap = fabs(sub) > fabs(ai);
      double piv = swap ? sub : ai;
      if (fabs(piv) < tol) piv = (piv < 0.0) ? -tol : tol;
      const double pinv = 1.0 / piv;
      double mult, an, bn, brow;
      if (swap) { mult = ai * pinv; brow = nd; an = bi - mult * nd; bn = -mult * ns; }
      else      { mult = sub * pinv; brow = bi; an = nd - mult * bi; bn = ns; }
      fa[base + (int64_t)r * nv] = pinv;
      fb[base + (int64_t)r * nv] = brow;
      fc[base + (int64_t)r * nv] = mult;
      fp[base + (int64_t)r * nv] = swap ? 1 : 0;
      ai = an; bi = bn;
    }
    if (fabs(ai) < tol) ai = (ai < 0.0) ? -tol : tol;
    fa[base + (int64_t)be * nv] = 1.0 / ai;
    fb[base + (int64_t)be * nv] = 0.0;
    for (int r = 0; r < bs; ++r) Z[base + (int64_t)r * nv] = 0.0;
    for (int r = be + 1; r < N; ++r) Z[base + (int64_t)r * nv] = 0.0;
  } else {
    bs = blk[(c * nv + v) * 2]; be = blk[(c * nv + v) * 2 + 1];
  }
  double ssq = 0.0;
  for (int it = 0; it < iters; ++it) {
    // forward elimination with the stored interchanges
    const bool gen = (!refine && it == 0);
    const uint64_t seed = ((uint64_t)(c * 1315423911ull) ^ ((uint64_t)v << 32));
    double cur = gen ? hash_uniform(seed + (uint64_t)bs * 0x632BE59BD9B4E019ull) : Z[base + (int64_t)bs * nv];
    for (int r = bs; r < be; ++r) {
      const double nxt = gen ? hash_uniform(seed + (uint64_t)(r + 1) * 0x632BE59BD9B4E019ull)
                             : Z[base + (int64_t)(r + 1) * nv];
      const double m = fc[base + (int64_t)r * nv];
      if (fp[base + (int64_t)r * nv]) { Z[base + (int64_t)r * nv] = nxt; cur = cur - m * nxt; }
      else { Z[base + (int64_t)r * nv] = cur; cur = nxt - m * cur; }
    }
    // back substitution (U has two super-diagonals; the second is e[r+1] on swapped rows)
    double x1 = cur * fa[base + (int64_t)be * nv], x2 = 0.0;
    ssq = x1 * x1;
    Z[base + (int64_t)be * nv] = x1;
    for (int r = be - 1; r >= bs; --r) {
      const double d2 = (fp[base + (int64_t)r * nv] && r + 1 < be) ? e[r + 1] : 0.0;
      const double x0 = (Z[base + (int64_t)r * nv] - fb[base + (int64_t)r * nv] * x1 - d2 * x2) * fa[base + (int64_t)r * nv];
      Z[base + (int64_t)r * nv] = x0;
      ssq += x0 * x0;
      x2 = x1; x1 = x0;
    }
    if (it + 1 < iters && ssq > 1e200) {   // guard against overflow on the next solve
      const double sc = rsqrt(ssq);
      for (int r = bs; r <= be; ++r) Z[base + (int64_t)r * nv] *= sc;
    }
  }
  const double sc = (ssq > 0.0) ? 1.0 / sqrt(ssq) : 0.0;
  for (int r = bs; r <= be; ++r) Z[base + (int64_t)r * nv] *= sc;
}

// Z [N][nv] real  ->  X [nv][N] complex (column-major N x nv frame), through a shared tile.
__global__ void k_z2x(const double* __restrict__ Z, cplx* __restrict__ X, int N, int nv, int tr, int tv) {
  __shared__ double tile[32][33];
  const int64_t c = blockIdx.x / (tr * tv);
  const int t = blockIdx.x % (tr * tv);
  const int r0 = (t % tr) * 32, v0 = (t / tr) * 32;
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;   // 32 x 8
  for (int q = ty; q < 32; q += 8) {
    const int r = r0 + q, v = v0 + tx;
    tile[q][tx] = (r < N && v < nv) ? Z[c * (int64_t)N * nv + (int64_t)r * nv + v] : 0.0;
  }
  __syncthreads();
  for (int q = ty; q < 32; q += 8) {
    const int v = v0 + q, r = r0 + tx;
    if (r < N && v < nv) X[c * (int64_t)N * nv + (int64_t)v * N + r] = mkc(tile[tx][q], 0.0);
  }
}

// Vbuf[(r - p - 1) + cc * N] = conj(V[r][cc]) for the WY block starting at column p (kb columns):
// zero above the unit diagonal, 1 on it, conj(B[r][p+cc]) below.  Also tauc = conj(tau).
__global__ void k_extract_v(const cplx* __restrict__ Bw, const cplx* __restrict__ tau, cplx* __restrict__ Vb,
                            cplx* __restrict__ tauc, int N, int p, int kb, int off) {
  const int64_t c = blockIdx.x;
  const cplx* B = Bw + c * (int64_t)N * N;
  cplx* V = Vb + c * (int64_t)N * NBT;
  const int rows = N - p - off;   // off = 1: tridiagonalization; off = KB: band reduction (heads KB below the diagonal)
  for (int idx = threadIdx.x; idx < rows * kb; idx += blockDim.x) {
    const int cc = idx / rows, rr = idx % rows;
    const int r = p + off + rr;
    cplx v;
    if (rr < cc) v = mkc(0.0, 0.0);
    else if (rr == cc) v = mkc(1.0, 0.0);
    else v = cconj(B[r + (int64_t)(p + cc) * N]);
    V[rr + (int64_t)cc * N] = v;
  }
  if (threadIdx.x < kb) tauc[c * NBT + threadIdx.x] = cconj(tau[c * N + p + threadIdx.x]);
}

// zlarft (forward, columnwise) from G = V^H V by recursive doubling: for a block [T11 T12; 0 T22]
// of two finished halves, T12 = -T11 G12 T22.  Starting from T_jj = tau_j the block size doubles
// log2(NBT) times; every level is two small matrix products done by all 1024 threads (element per
// thread), instead of NBT dependent column solves by NBT threads.  T, G column-major, ld NBT;
// tmp holds T11 G12.  Rows / columns >= kb are zero (G is not defined there).
__global__ void __launch_bounds__(1024) k_larft(const cplx* __restrict__ G, const cplx* __restrict__ tauc,
                                                cplx* __restrict__ T, cplx* __restrict__ tmp, int kb) {
  const int64_t c = blockIdx.x;
  const cplx* g = G + c * NBT * NBT;
  cplx* t = T + c * NBT * NBT;
  cplx* w = tmp + c * NBT * NBT;
  const int tid = threadIdx.x, nt = blockDim.x;
  int kbp = 1;
  while (kbp < kb) kbp <<= 1;               // only the leading kbp x kbp part is built (kb <= kbp <= NBT)
  for (int idx = tid; idx < kbp * kbp; idx += nt) {
    const int r = idx % kbp, cc = idx / kbp;
    t[r + cc * NBT] = (r == cc && r < kb) ? tauc[c * NBT + r] : mkc(0.0, 0.0);
  }
  __syncthreads();
  for (int sz = 1; sz < kbp; sz <<= 1) {
    // tmp[r][cc] = sum_q T11[r][q] G[q][cc]: r, q in the first half (q >= r), cc in the second half
    const int per = sz * sz, pairs = kbp / (2 * sz);
    for (int idx = tid; idx < per * pairs; idx += nt) {
      const int b0 = (idx / per) * 2 * sz, e = idx % per;
      const int r = b0 + e % sz, cc = b0 + sz + e / sz;
      cplx acc = mkc(0.0, 0.0);
      if (cc < kb)
        for (int q = r; q < b0 + sz && q < kb; ++q) cfma(acc, t[r + q * NBT], g[q + cc * NBT]);   // G is defined for q < kb only
      w[r + cc * NBT] = acc;
    }
    __syncthreads();
    // T12[r][cc] = -sum_q tmp[r][q] T22[q][cc]: q, cc in the second half (q <= cc)
    for (int idx = tid; idx < per * pairs; idx += nt) {
      const int b0 = (idx / per) * 2 * sz, e = idx % per;
      const int r = b0 + e % sz, cc = b0 + sz + e / sz;
      cplx acc = mkc(0.0, 0.0);
      if (cc < kb)
        for (int q = b0 + sz; q <= cc; ++q) cfma(acc, w[r + q * NBT], t[q + cc * NBT]);
      t[r + cc * NBT] = mkc(-acc.x, -acc.y);
    }
    __syncthreads();
  }
}

__global__ void k_set_info(int* info, int64_t cnt) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i < cnt) info[i] = 0;
}

// transpose-convert frames X [cnt][nv][N] -> public layout U [cnt][N][nv]
__global__ void k_x2u(const cplx* __restrict__ X, cplx* __restrict__ U, int N, int nv, int tr, int tv) {
  __shared__ cplx tile[32][33];
  const int64_t c = blockIdx.x / (tr * tv);
  const int t = blockIdx.x % (tr * tv);
  const int r0 = (t % tr) * 32, v0 = (t / tr) * 32;
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
  for (int q = ty; q < 32; q += 8) {
    const int v = v0 + q, r = r0 + tx;
    tile[q][tx] = (r < N && v < nv) ? X[c * (int64_t)N * nv + (int64_t)v * N + r] : mkc(0.0, 0.0);
  }
  __syncthreads();
  for (int q = ty; q < 32; q += 8) {
    const int r = r0 + q, v = v0 + tx;
    if (r < N && v < nv) U[c * (int64_t)N * nv + (int64_t)r * nv + v] = tile[tx][q];
  }
}

}  // namespace

// scratch layout for ``cnt`` matrices
struct EighScratch {
  cplx *Bw, *Wp, *P, *zpart, *tau, *Vb, *T, *G, *tauc, *Y, *Y2, *pq, *Ttmp;
  double *d, *e, *tnorm, *Z, *fa, *fb, *fc;
  unsigned char* fp;
  int* blk;
  double *blo, *bhi;
  int* bcl;
  void* orth;
  int* hcount;
  void* band;
};

static size_t eigh_large_carve(char* base, int64_t cnt, int N, int nv, EighScratch* s) {
  size_t off = 0;
  auto take = [&](size_t bytes) { char* p = base ? base + off : nullptr; off += be_align256(bytes); return p; };
  const int nJmax = (N + HB - 1) / HB;
  const size_t nn = (size_t)N * N, nvN = (size_t)N * (nv > 0 ? nv : 1);
  cplx* Bw = (cplx*)take(cnt * nn * sizeof(cplx));
  cplx* Wp = (cplx*)take(cnt * (size_t)N * NB * sizeof(cplx));
  cplx* P = (cplx*)take(cnt * (size_t)nJmax * N * sizeof(cplx));
  cplx* zp = (cplx*)take(cnt * (size_t)N * sizeof(cplx));
  cplx* tau = (cplx*)take(cnt * (size_t)N * sizeof(cplx));
  cplx* Vb = (cplx*)take(cnt * (size_t)N * NBT * sizeof(cplx));
  cplx* T = (cplx*)take(cnt * (size_t)NBT * NBT * sizeof(cplx));
  cplx* G = (cplx*)take(cnt * (size_t)NBT * NBT * sizeof(cplx));
  cplx* tauc = (cplx*)take(cnt * (size_t)NBT * sizeof(cplx));
  cplx* Y = (cplx*)take(cnt * (size_t)NBT * (nv > 0 ? nv : 1) * sizeof(cplx));
  cplx* Y2 = (cplx*)take(cnt * (size_t)NBT * (nv > 0 ? nv : 1) * sizeof(cplx));
  cplx* pq = (cplx*)take(cnt * (size_t)2 * NB * sizeof(cplx));
  cplx* Ttmp = (cplx*)take(cnt * (size_t)NBT * NBT * sizeof(cplx));
  double* d = (double*)take(cnt * (size_t)N * sizeof(double));
  double* e = (double*)take(cnt * (size_t)N * sizeof(double));
  double* tn = (double*)take(cnt * sizeof(double));
  double* Z = (double*)take(cnt * nvN * sizeof(double));
  double* fa = (double*)take(cnt * nvN * sizeof(double));
  double* fb = (double*)take(cnt * nvN * sizeof(double));
  double* fc = (double*)take(cnt * nvN * sizeof(double));
  unsigned char* fp = (unsigned char*)take(cnt * nvN);
  int* blk = (int*)take(cnt * (size_t)(nv > 0 ? nv : 1) * 2 * sizeof(int));
  double* blo = (double*)take(cnt * (size_t)N * sizeof(double));
  double* bhi = (double*)take(cnt * (size_t)N * sizeof(double));
  int* bcl = (int*)take(cnt * (size_t)N * sizeof(int));
  void* orth = take(be_cluster_orth_scratch_bytes(cnt, N, nv));
  int* hcount = (int*)take((size_t)N * sizeof(int));
  void* band = (N >= BE_BAND_MINN && N <= BE_BAND_MAXN) ? take(be_band_scratch_bytes(cnt, N)) : nullptr;
  if (s) { *s = EighScratch{Bw, Wp, P, zp, tau, Vb, T, G, tauc, Y, Y2, pq, Ttmp, d, e, tn, Z, fa, fb, fc, fp, blk, blo, bhi, bcl, orth, hcount, band}; }
  return off;
}

size_t be_eigh_large_scratch_bytes(int64_t cnt, int N, int nv) { return eigh_large_carve(nullptr, cnt, N, nv, nullptr); }

#define LAUNCH_CHECK() do { ctx->launches++; cudaError_t e__ = cudaGetLastError(); if (e__ != cudaSuccess) return (int)e__; } while (0)

int be_eigh_large(be_ctx* ctx, const cplx* H, const GridMap& map, int64_t loop0, int64_t cnt, int N,
                  int nv, int ne, double* E, cplx* X, int* info) {
  if (ne < nv) ne = nv;
  if (ne > N) ne = N;
  const size_t need = be_eigh_large_scratch_bytes(cnt, N, nv);
  char* base = (char*)be_arena_alloc(ctx, need);
  if (!base) return BE_ERR_NOMEM;
  EighScratch s;
  eigh_large_carve(base, cnt, N, nv, &s);
  cudaStream_t st = ctx->stream;
  if (cnt > 0x7fffffffLL / 64) return BE_ERR_SHAPE;
  const int nJmax = (N + HB - 1) / HB;

  if (info) { k_set_info<<<(unsigned)((cnt + 255) / 256), 256, 0, st>>>(info, cnt); LAUNCH_CHECK(); }
  const bool on_chip = N <= TS_MAXN;   // whole matrix in one CTA's shared memory (tridiag_small.cu)
  if (on_chip) {
    BE_TRY(be_tridiag_small(ctx, H, map, loop0, cnt, N, s.Bw, s.d, s.e, s.tau));
  } else if (ctx->bloch) {
    BE_TRY(be_bloch_assemble_chunk(ctx, ctx->bloch, loop0, cnt, N, s.Bw));   // H(k) generated into the work copy
  } else if (!ctx->feed) {
    const int nchunk = (int)(((int64_t)N * N + 2047) / 2048);
    k_gather<<<(unsigned)(cnt * nchunk), 256, 0, st>>>(H, s.Bw, map, loop0, N, nchunk);
    LAUNCH_CHECK();
  }
  const size_t ysh_bytes = 2 * (size_t)N * sizeof(cplx);
  if (ysh_bytes > 200 * 1024) return BE_ERR_UNSUPPORTED;
  if (ysh_bytes > 48 * 1024) BE_CUDA(cudaFuncSetAttribute(k_colw, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ysh_bytes));
  BE_CUDA(cudaFuncSetAttribute(k_hemv, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)HEMV_SMEM));
  auto colw = [&](int i, int p, int do_w, int do_col) {
    const int n = N - i - 1, kk = i - p;
    be_prof_begin(ctx, PK_COL);
    k_colw<<<(unsigned)cnt, CW_THREADS, ysh_bytes, st>>>(s.Bw, s.Wp, s.P, s.zpart, s.pq, s.d, s.e, s.tau, N, i, p,
                                                         nJmax, do_w, do_col);
    // panels V, W read once (2 kk columns), y partials, v, w out, column in / out
    be_prof_end(ctx, PK_COL, (double)cnt * (n + 1) * 16.0 * (2.0 * kk + 6.0 + 0.5 * ((n + HB - 1) / HB)),
                (double)cnt * (n + 1) * 32.0 * kk);
  };

  // ---- S1a: blocked tridiagonalization
  BE_CUDA(cudaMemsetAsync(s.hcount, 0, (size_t)N * sizeof(int), st));   // work counters of the persistent k_hemv, one per column
  // panel width: the panel work (k_colw and the panel block columns of k_hemv) grows with nb / n, the
  // rank-2k GEMM likes a deep K = 2 nb: 16 for mid-size matrices, NB = 32 for large ones
  const int nb = (N <= 640) ? NB / 2 : NB;
  // 1: two-stage wherever it is supported; 2 (default): where it is faster -- measured on B200: N = 1600 (half of the
  // vectors) 905 vs 1035 ms per 300 matrices, N = 800 (all vectors) 215 vs 203 ms, N = 400 even
  const bool two_stage = N >= BE_BAND_MINN && N <= BE_BAND_MAXN &&
                         (ctx->eigh_algo == 1 || (ctx->eigh_algo == 2 && N >= BE_BAND_AUTON));
  if (ctx->feed) {
    // host grid streamed into this chunk (HostFeed, be_common.cuh): gather sub-range j when its copy has landed,
    // hand the staging buffer back, and reduce the sub-range to band form while the next one travels
    HostFeed* f = ctx->feed;
    ctx->feed = nullptr;
    if (!two_stage || f->mstart[f->nsub] != cnt) return BE_ERR_UNSUPPORTED;   // the caller checks both
    GridMap fm;
    memset(&fm, 0, sizeof(fm));
    fm.ndim = 1; fm.dir = 0; fm.n1 = 1; fm.dims[0] = 1; fm.batch_stride = 1;
    const int nchunk = (int)(((int64_t)N * N + 2047) / 2048);
    for (int j = 0; j < f->nsub; ++j) {
      const int64_t c0 = f->mstart[j], cs = f->mstart[j + 1] - c0;
      fm.loops = cs;
      BE_CUDA(cudaStreamWaitEvent(st, f->copied[j & 1], 0));
      k_gather<<<(unsigned)(cs * nchunk), 256, 0, st>>>((const cplx*)f->buf[j & 1], s.Bw + c0 * (int64_t)N * N, fm, 0, N, nchunk);
      LAUNCH_CHECK();
      BE_CUDA(cudaEventRecord(f->freed[j & 1], st));
      if (j + 2 < f->nsub) BE_TRY(f->issue(f->self, j + 2));
      BE_TRY(be_band_stage1(ctx, s.Bw + c0 * (int64_t)N * N, cs, N, s.tau + c0 * N, s.band));
    }
    BE_TRY(be_band_stage2(ctx, s.Bw, cnt, N, s.d, s.e, s.band));
  } else if (two_stage) {
    BE_TRY(be_band_reduce(ctx, s.Bw, cnt, N, s.d, s.e, s.tau, s.band));
  }
  for (int p = 0; p < N && !on_chip && !two_stage; p += nb) {
    if (p > 0 && N - p <= TS_MAXN) {
      // the trailing block is up to date at a panel boundary and fits one CTA's shared memory: its ~100
      // columns are too short to feed two launches each (k_hemv bottoms out at ~50 us per launch)
      BE_TRY(be_tridiag_small(ctx, nullptr, map, loop0, cnt, N, s.Bw, s.d, s.e, s.tau, p));
      break;
    }
    const int pend = (p + nb < N - 1) ? p + nb : N - 1;   // reflector columns p .. pend-1
    colw(p, p, 0, 1);   // reflector of column p (or, when p == N-1, just the last diagonal entry)
    LAUNCH_CHECK();
    if (p >= N - 1) break;
    for (int i = p; i < pend; ++i) {
      const int n = N - i - 1;
      const int nJ = (n + HB - 1) / HB;
      const int npb = (2 * (i - p) + HB - 1) / HB;   // panel blocks: the 2k dot products for k_colw
      be_prof_begin(ctx, PK_HEMV);
      {
        const int64_t total = cnt * (int64_t)(nJ + npb);
        const int64_t grid = total < 2 * (int64_t)ctx->sm_count ? total : 2 * (int64_t)ctx->sm_count;
        k_hemv<<<(unsigned)grid, HEMV_THREADS, HEMV_SMEM, st>>>(s.Bw, s.P, s.zpart, N, i, nJ, nJmax, s.Wp, s.pq, p, npb,
                                                                 s.hcount + i, (int)total);
      }
      // algorithmic traffic: the lower triangle once, v in, y out; 8 real flops per complex fma, 2 per element
      be_prof_end(ctx, PK_HEMV, (double)cnt * (0.5 * n * (n + 1.0) + 2.0 * n) * 16.0, (double)cnt * 8.0 * n * n);
      LAUNCH_CHECK();
      colw(i, p, 1, (i + 1 < pend) ? 1 : 0);   // w_i, and the reflector of column i+1 inside the panel
      LAUNCH_CHECK();
    }
    const int q = pend, kb = pend - p;
    if (q < N) {
      const int n2 = N - q;
      // B[q:, q:] -= [V W] [W V]^H  (lower tiles): one rank-2kb update, the two K segments read in place
      ZgemmParams g = zgemm_simple(n2, n2, 2 * kb, s.Bw + q + (int64_t)p * N, N, (int64_t)N * N,
                                   s.Wp + q, N, (int64_t)N * NB,
                                   s.Bw + q + (int64_t)q * N, N, (int64_t)N * N, cnt);
      g.A2 = s.Wp + q; g.sA2o = (int64_t)N * NB;
      g.B2 = s.Bw + q + (int64_t)p * N; g.sB2o = (int64_t)N * N;
      g.ksplit = kb;
      g.alpha = mkc(-1.0, 0.0); g.beta = mkc(1.0, 0.0); g.lower = 1;
      BE_TRY(be_zgemm(ctx, BE_OP_N, BE_OP_C, g));
    }
    if (pend == N - 1) {   // last diagonal element (no pending panel: it was just applied)
      colw(N - 1, N - 1, 0, 1);
      LAUNCH_CHECK();
      break;
    }
  }

  if (ctx->split_after_tridiag) {
    // chunk pipeline: the rest of this chunk continues on the second stream, the caller's next
    // chunk starts its tridiagonalization on the first one
    ctx->split_after_tridiag = 0;
    BE_CUDA(cudaEventRecord(ctx->ev_split, st));
    BE_CUDA(cudaStreamWaitEvent(ctx->stream2, ctx->ev_split, 0));
    ctx->stream = ctx->stream2;
    st = ctx->stream2;
  }

  // ---- S1b: tridiagonal eigenproblem
  {
    const int nblk = (ne + 127) / 128;
    const size_t sh = 2 * (size_t)N * sizeof(double);
    if (sh > 48 * 1024) {
      BE_CUDA(cudaFuncSetAttribute(k_bisect, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sh));
      BE_CUDA(cudaFuncSetAttribute(k_invit, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sh));
    }
    be_prof_begin(ctx, PK_BISECT);
    const int mpb = ne <= 64 ? 128 / ne : 1;
    if (mpb > 1 && 3 * (size_t)mpb * N * sizeof(double) <= 48 * 1024)
      k_bisect_packed<<<(unsigned)((cnt + mpb - 1) / mpb), 128, 3 * (size_t)mpb * N * sizeof(double), st>>>(
          s.d, s.e, E, s.tnorm, s.blo, s.bhi, s.bcl, N, cnt, ne, mpb);
    else
      k_bisect<<<(unsigned)(cnt * nblk), 128, sh, st>>>(s.d, s.e, E, s.tnorm, s.blo, s.bhi, s.bcl, N, nblk, ne);
    be_prof_end(ctx, PK_BISECT, (double)cnt * N * 24.0, 0.0);
    LAUNCH_CHECK();
    if (nv > 0) {
      const int nvb = (nv + 127) / 128;
      // Inverse iteration, one solve at a time with the clusters re-orthogonalized after every solve
      // (subspace iteration inside a cluster): several solves in a row with the SAME shift collapse
      // the vectors of a numerically degenerate cluster onto its few nearest eigen-directions
      // (measured: cond 6e10 for the 400-fold +-1 of the projected spin operator).
      const int nsolve = ctx->invit_solves < 1 ? 1 : ctx->invit_solves;
      for (int it = 0; it < nsolve; ++it) {
        be_prof_begin(ctx, PK_INVIT);
        k_invit<<<(unsigned)(cnt * nvb), 128, sh, st>>>(s.d, s.e, E, s.tnorm, s.fa, s.fb, s.fc, s.fp, s.blk, s.blo, s.bhi,
                                                        s.bcl, s.Z, N, nv, nvb, it > 0 ? 1 : 0, 1);
        be_prof_end(ctx, PK_INVIT, (double)cnt * N * nv * 8.0, 0.0);
        LAUNCH_CHECK();
        // Cholesky-QR passes: 2 after the first solve (random starts: cond up to ~1e5) and after the last
        // one (final orthogonality at eps); 1 in between (one solve applied to an orthonormal basis keeps
        // cond below ~5e2, and the next solve re-mixes the cluster anyway)
        BE_TRY(be_cluster_orth(ctx, E, s.tnorm, s.blk, s.Z, cnt, N, nv, CLUSTER_TOL, info, s.orth, it == 0,
                               (it == 0 || it == nsolve - 1) ? 2 : 1));
      }
    }
  }
  if (nv == 0) return BE_OK;

  // ---- S1c: back-transform X = conj(Q) Z: on chip for small matrices, else compact-WY blocks, last block first
  if (on_chip) return be_backtransform_small(ctx, s.Bw, s.tau, s.Z, X, cnt, N, nv);
  {
    const int tr = (N + 31) / 32, tv = (nv + 31) / 32;
    k_z2x<<<(unsigned)(cnt * tr * tv), 256, 0, st>>>(s.Z, X, N, nv, tr, tv);
    LAUNCH_CHECK();
  }
  // two-stage: first the short reflectors of the bulge chasing, then the band reduction's reflectors, whose
  // heads sit KB rows below the diagonal (columns 0 .. N - KB - 1)
  if (two_stage) BE_TRY(be_band_q2(ctx, s.Bw, X, cnt, N, nv));
  const int off = two_stage ? BE_BAND_KB : 1;
  const int nref = N - off;
  int plast = ((nref - 1) / NBT) * NBT;
  for (int p = plast; p >= 0; p -= NBT) {
    const int pend = (p + NBT < nref) ? p + NBT : nref;
    const int kb = pend - p;
    if (kb <= 0) continue;
    const int rows = N - p - off;
    k_extract_v<<<(unsigned)cnt, 256, 0, st>>>(s.Bw, s.tau, s.Vb, s.tauc, N, p, kb, off);
    LAUNCH_CHECK();
    // G = V^H V
    ZgemmParams gg = zgemm_simple(kb, kb, rows, s.Vb, N, (int64_t)N * NBT, s.Vb, N, (int64_t)N * NBT,
                                  s.G, NBT, NBT * NBT, cnt);
    BE_TRY(be_zgemm(ctx, BE_OP_C, BE_OP_N, gg));
    k_larft<<<(unsigned)cnt, kb <= 64 ? 256 : 1024, 0, st>>>(s.G, s.tauc, s.T, s.Ttmp, kb);
    LAUNCH_CHECK();
    // Y = V^H X[p+1:, :]
    ZgemmParams gy = zgemm_simple(kb, nv, rows, s.Vb, N, (int64_t)N * NBT, X + p + off, N, (int64_t)N * nv,
                                  s.Y, NBT, (int64_t)NBT * nv, cnt);
    BE_TRY(be_zgemm(ctx, BE_OP_C, BE_OP_N, gy));
    // Y2 = T Y
    ZgemmParams gt = zgemm_simple(kb, nv, kb, s.T, NBT, NBT * NBT, s.Y, NBT, (int64_t)NBT * nv,
                                  s.Y2, NBT, (int64_t)NBT * nv, cnt);
    BE_TRY(be_zgemm(ctx, BE_OP_N, BE_OP_N, gt));
    // X[p+1:, :] -= V Y2
    ZgemmParams gx = zgemm_simple(rows, nv, kb, s.Vb, N, (int64_t)N * NBT, s.Y2, NBT, (int64_t)NBT * nv,
                                  X + p + off, N, (int64_t)N * nv, cnt);
    gx.alpha = mkc(-1.0, 0.0); gx.beta = mkc(1.0, 0.0);
    BE_TRY(be_zgemm(ctx, BE_OP_N, BE_OP_N, gx));
  }
  return BE_OK;
}

// public-layout conversion used by be_eigh_batched
int be_frames_to_public(be_ctx* ctx, const cplx* X, cplx* U, int64_t cnt, int N, int nv) {
  const int tr = (N + 31) / 32, tv = (nv + 31) / 32;
  if (cnt * tr * tv > 0x7fffffffLL) return BE_ERR_SHAPE;
  k_x2u<<<(unsigned)(cnt * tr * tv), 256, 0, ctx->stream>>>(X, U, N, nv, tr, tv);
  LAUNCH_CHECK();
  return BE_OK;
}
