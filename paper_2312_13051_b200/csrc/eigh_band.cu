// S1a, two-stage variant -- Hermitian tridiagonalization without a level-2 pass over the trailing matrix
// ("exact diagonalization ... at many points in reciprocal space" is where the time goes;
// SURVEY 7.3 H1 names the two-stage reduction as the fallback when the HEMV half of the one-stage
// reduction caps the total).
//
//   stage 1  dense -> band of width KB = 8:  B = Q1 A_band Q1^H.  Per panel of KB columns
//              k_ysum, k_wupd : wide kernels -- sum the partial products of the previous panel (Y = A V), finish
//                        W = Y T - V C and bring the next KB columns up to date
//              k_panel : one CTA per matrix -- Householder QR of those columns below the band (one block
//                        reduction per column), explicit V panel for the streaming kernel
//              k_fused : ONE streaming pass over the trailing matrix per panel: every 64 x 64 tile is read
//                        once (TMA bulk copies), gets the pending rank-2KB update of the previous panel
//                        A -= W V^H + V W^H on the FP64 tensor cores, is written back (bulk store), and is
//                        multiplied by the new panel's V from both sides of the symmetry (Y = A V) before
//                        it leaves the SM.  16 flops per byte of HBM traffic instead of the 1 flop per
//                        byte of a HEMV.
//   stage 2  band -> real tridiagonal by bulge chasing (k_chase4): one CTA per matrix, eight lanes per sweep,
//            sweeps pipelined two chase steps apart, the band window in a shared-memory ring; the reflectors
//            (length KB) go to the unused upper triangle of the work matrix.
//   Q2       X <- conj(Q2) X (k_q2): the N^2 / (2 KB) short reflectors are applied with the eigenvector
//            entries in registers: a thread owns one column and a sliding window of QG + KB - 1 rows, a
//            group of QG consecutive sweeps is applied per pass over the column (plain DFMA: on B200 the
//            DMMA and DFMA peaks are equal, and the diamond-shaped WY form of these reflectors would
//            cost 2-4x their flops).
//   Q1       compact-WY GEMMs of the one-stage path (eigh_large.cu) with the reflector heads KB rows
//            below the diagonal.
//
// Memory view as in eigh_large.cu: B = conj(H) column-major, lower triangle referenced; the upper
// triangle of the diagonal tiles is kept as the mirror image during stage 1 so that a diagonal tile is an
// ordinary full tile for the multiplication.
#include "be_common.cuh"
#include "tma.cuh"
#include <float.h>
#include <vector>

namespace {

constexpr int KB = BE_BAND_KB;     // band width
constexpr int LDR = 65;            // shared-memory stride of a panel column in k_fused (= 1 mod 4: conflict-free fragment loads)
constexpr int TS = 64;             // tile of the streaming kernel
constexpr int LDT = 67;            // shared-memory column stride of a tile (= 3 mod 8)
constexpr int LDAB = 2 * KB;       // compact band storage: AB[j][d] = A[j + d][j], d < 2 KB (bulge included)

__device__ __forceinline__ void dmma(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}
__device__ __forceinline__ cplx shfl_c(cplx v, int src) {
  return mkc(__shfl_sync(0xffffffffu, v.x, src), __shfl_sync(0xffffffffu, v.y, src));
}
__device__ __forceinline__ cplx shfl_xor_c(cplx v, int m) {
  return mkc(__shfl_xor_sync(0xffffffffu, v.x, m), __shfl_xor_sync(0xffffffffu, v.y, m));
}

// Scalars of a Householder reflector H = I - tau v v^H, H^H (alpha; x) = (beta; 0), |x|^2 = xn2 > 0 or Im alpha != 0
// (zlarfg): beta = -sign(Re alpha) sqrt(|alpha|^2 + xn2), tau = (beta - alpha) / beta, v = x / (alpha - beta).
// IEEE double division and square root are ~100-instruction dependent chains on the GPU, and these scalars sit on
// the critical path of every chase step and every panel column: rsqrt + one Newton step and one reciprocal instead.
__device__ __forceinline__ void larfg_scalars(cplx alpha, double xn2, double& beta, cplx& tau, cplx& scale) {
  const double s2 = cabs2(alpha) + xn2;
  const double r = rsqrt(s2);
  double nb = s2 * r;
  nb = fma(0.5 * r, fma(-nb, nb, s2), nb);          // |beta| to the last bit or two
  const bool pos = alpha.x >= 0.0;
  beta = pos ? -nb : nb;
  const double ib = pos ? -r : r;                    // 1 / beta (relative error ~1e-16)
  tau = mkc(fma(-alpha.x, ib, 1.0), -alpha.y * ib);
  const double dx = alpha.x - beta;                  // no cancellation: beta has the opposite sign
  const double rd = __drcp_rn(fma(dx, dx, alpha.y * alpha.y));
  scale = mkc(dx * rd, -alpha.y * rd);
}

// ------------------------------------------------------------------------------------------
// The diagonal 64 x 64 tiles get their upper triangle from the lower one (the input contract reads
// only one triangle of H), and an exactly real diagonal.
__global__ void k_symdiag(cplx* __restrict__ Bw, int N) {
  const int c0 = blockIdx.x * TS;
  cplx* B = Bw + (int64_t)blockIdx.y * N * N;
  for (int idx = threadIdx.x; idx < TS * TS; idx += blockDim.x) {
    const int rr = idx % TS, cc = idx / TS;
    const int r = c0 + rr, col = c0 + cc;
    if (r >= N) continue;
    if (rr > cc) B[col + (int64_t)r * N] = cconj(B[r + (int64_t)col * N]);
    else if (rr == cc) B[r + (int64_t)r * N].y = 0.0;
  }
}

// ------------------------------------------------------------------------------------------
// Block-wide sum of KB complex values per thread (PT threads); result in res[0..KB).
constexpr int PT = 512;
__device__ __forceinline__ void block_sum8(const cplx (&part)[KB], cplx* red, cplx* res) {
  static_assert(KB == 8, "butterfly written for 8 values");
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const bool u16 = lane & 16, u8 = lane & 8, u4 = lane & 4;
  cplx b4[4], b2[2], b1;
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    const cplx snd = u16 ? part[j] : part[j + 4], kp = u16 ? part[j + 4] : part[j];
    b4[j] = cadd(kp, shfl_xor_c(snd, 16));
  }
#pragma unroll
  for (int j = 0; j < 2; ++j) {
    const cplx snd = u8 ? b4[j] : b4[j + 2], kp = u8 ? b4[j + 2] : b4[j];
    b2[j] = cadd(kp, shfl_xor_c(snd, 8));
  }
  {
    const cplx snd = u4 ? b2[0] : b2[1], kp = u4 ? b2[1] : b2[0];
    b1 = cadd(kp, shfl_xor_c(snd, 4));
  }
  b1 = cadd(b1, shfl_xor_c(b1, 2));
  b1 = cadd(b1, shfl_xor_c(b1, 1));
  if ((lane & 3) == 0) red[warp * KB + (u16 ? 4 : 0) + (u8 ? 2 : 0) + (u4 ? 1 : 0)] = b1;
  __syncthreads();
  if (threadIdx.x < KB) {
    cplx t = mkc(0.0, 0.0);
#pragma unroll
    for (int w = 0; w < PT / 32; ++w) t = cadd(t, red[w * KB + threadIdx.x]);
    res[threadIdx.x] = t;
  }
  __syncthreads();
}

// Explicit panels (V of the new panel, V and W of the previous one) and the partial products are stored
// column by column: element (row r, panel column q) of matrix c at ((c KB + q) Np + r), Np = rows padded to
// whole tiles.  Rows above the panel's first row and beyond N hold exact zeros.
#define PIX(q, r) ((int64_t)(q) * Np + (r))

// Y = A V of panel p-1 from the partial products of k_fused (row parts per block column J <= I, column part
// Zc), one CTA per (row tile I, matrix); thread = (row, q).  Also the tile's share of M = V^H Y, summed by k_wupd.
__global__ void __launch_bounds__(512) k_ysum(const cplx* __restrict__ P, const cplx* __restrict__ Zc,
                                              const cplx* __restrict__ Vprev, cplx* __restrict__ Wx, cplx* __restrict__ Mpart,
                                              int N, int Np, int nT, int J0, int jprev) {
  __shared__ cplx Ysh[TS * KB], Vsh[TS * KB], Msh[8 * 64];
  const int64_t c = blockIdx.y;
  const int I = J0 + blockIdx.x;
  const int tid = threadIdx.x, q = tid >> 6, rl = tid & 63;
  const int r = I * TS + rl;
  cplx y = mkc(0.0, 0.0), v = mkc(0.0, 0.0);
  if (r >= jprev && r < N) {
    y = Zc[c * KB * (int64_t)Np + PIX(q, r)];
    const cplx* pp = P + (c * nT + J0) * (int64_t)KB * Np + PIX(q, r);
    int J = J0;
    for (; J + 4 <= I + 1; J += 4) {
      const cplx p0 = pp[0], p1 = pp[(int64_t)KB * Np], p2 = pp[2 * (int64_t)KB * Np], p3 = pp[3 * (int64_t)KB * Np];
      y = cadd(cadd(y, cadd(p0, p1)), cadd(p2, p3));
      pp += 4 * (int64_t)KB * Np;
    }
    for (; J <= I; ++J) { y = cadd(y, pp[0]); pp += (int64_t)KB * Np; }
    v = Vprev[c * KB * (int64_t)Np + PIX(q, r)];
  }
  Wx[c * KB * (int64_t)Np + PIX(q, r)] = y;
  Ysh[rl * KB + q] = y;
  Vsh[rl * KB + q] = v;
  __syncthreads();
  {
    const int pid = tid & 63, slice = tid >> 6, mq = pid >> 3, mq2 = pid & 7;
    cplx macc = mkc(0.0, 0.0);
#pragma unroll
    for (int rr = slice * 8; rr < slice * 8 + 8; ++rr) cfmac(macc, Vsh[rr * KB + mq], Ysh[rr * KB + mq2]);
    Msh[slice * 64 + pid] = macc;
  }
  __syncthreads();
  if (tid < 64) {
    cplx t = mkc(0.0, 0.0);
#pragma unroll
    for (int sl = 0; sl < 8; ++sl) t = cadd(t, Msh[sl * 64 + tid]);
    Mpart[(c * nT + I) * 64 + tid] = t;
  }
}

// Per-matrix scalars of a panel step (p > 0), one small CTA per matrix: M = sum of the tiles' shares of V^H Y,
// C = 1/2 T^H M T, and the top KB + 1 rows of V and of W = Y T - V C (every row of the column update needs them).
// Layout of MC [cnt][64 + 2 * 72]: C, Vtop [9][8], Wtop [9][8].
constexpr int MC_STRIDE = 64 + 2 * (KB + 1) * KB;
__global__ void __launch_bounds__(96) k_mc(const cplx* __restrict__ Yx, const cplx* __restrict__ Vprev,
                                           const cplx* __restrict__ Mpart, const cplx* __restrict__ T1,
                                           cplx* __restrict__ MC, int N, int Np, int nT, int J0, int jprev) {
  __shared__ cplx Ts[KB * KB], Cs[KB * KB], Mf[64], Yt[(KB + 1) * KB], Vt[(KB + 1) * KB];
  const int64_t c = blockIdx.x;
  const int tid = threadIdx.x;
  const cplx* __restrict__ Y = Yx + c * KB * (int64_t)Np;
  const cplx* __restrict__ Vp = Vprev + c * KB * (int64_t)Np;
  if (tid < 64) {
    Ts[tid] = T1[c * 64 + tid];
    cplx t0 = mkc(0.0, 0.0), t1 = mkc(0.0, 0.0);
    int I2 = J0;
    for (; I2 + 1 < nT; I2 += 2) {   // independent loads
      t0 = cadd(t0, Mpart[(c * nT + I2) * 64 + tid]);
      t1 = cadd(t1, Mpart[(c * nT + I2 + 1) * 64 + tid]);
    }
    if (I2 < nT) t0 = cadd(t0, Mpart[(c * nT + I2) * 64 + tid]);
    Mf[tid] = cadd(t0, t1);
  }
  if (tid < (KB + 1) * KB) {
    const int tr = tid / KB, tq = tid % KB;
    const int rr = jprev + tr;
    Yt[tid] = (rr < N) ? Y[PIX(tq, rr)] : mkc(0.0, 0.0);
    Vt[tid] = (rr < N) ? Vp[PIX(tq, rr)] : mkc(0.0, 0.0);
  }
  __syncthreads();
  if (tid < 64) {
    const int a = tid >> 3, b2 = tid & 7;
    cplx acc = mkc(0.0, 0.0);
    for (int k2 = 0; k2 < KB; ++k2) {
      cplx t = mkc(0.0, 0.0);
      for (int k1 = 0; k1 < KB; ++k1) cfmac(t, Ts[k1 * KB + a], Mf[k1 * KB + k2]);   // conj(T[k1][a]) M[k1][k2]
      cfma(acc, t, Ts[k2 * KB + b2]);
    }
    Cs[tid] = cscale(0.5, acc);
    MC[c * MC_STRIDE + tid] = Cs[tid];
  }
  __syncthreads();
  if (tid < (KB + 1) * KB) {
    const int tr = tid / KB, tq = tid % KB;
    cplx w = mkc(0.0, 0.0);
#pragma unroll
    for (int k1 = 0; k1 < KB; ++k1) { cfma(w, Yt[tr * KB + k1], Ts[k1 * KB + tq]); cfms(w, Vt[tr * KB + k1], Cs[k1 * KB + tq]); }
    MC[c * MC_STRIDE + 64 + tid] = Vt[tid];
    MC[c * MC_STRIDE + 64 + (KB + 1) * KB + tid] = w;
  }
}

// Second wide kernel of a panel step (p > 0), one CTA per (row tile I, matrix), thread = (row, column):
//   W_{p-1} = Y T - V C for the rows of the tile  -> Wx (explicit panel for k_fused: zero above j2)
//   the columns p KB .. of the trailing matrix receive the pending update  -= W V^H + V W^H, in place
//   (ncol = KB columns; at the end of stage 1 the whole trailing block of at most KB + 1 columns).
__global__ void __launch_bounds__(512) k_wupd(cplx* __restrict__ Bw, const cplx* __restrict__ Yx, const cplx* __restrict__ Vprev,
                                              cplx* __restrict__ Wx, const cplx* __restrict__ MC,
                                              const cplx* __restrict__ T1, int N, int Np, int J0, int jprev, int ncol) {
  __shared__ cplx Ts[KB * KB], Cs[KB * KB], Vtop[(KB + 1) * KB], Wtop[(KB + 1) * KB];
  __shared__ cplx Ysh[TS * (KB + 1)], Vsh[TS * (KB + 1)], Wsh[TS * (KB + 1)];
  const int64_t c = blockIdx.y;
  const int I = J0 + blockIdx.x;
  const int tid = threadIdx.x, q = tid >> 6, rl = tid & 63;
  const int r = I * TS + rl, j2 = jprev + KB;
  cplx* __restrict__ B = Bw + c * (int64_t)N * N;
  if (tid < 64) { Ts[tid] = T1[c * 64 + tid]; Cs[tid] = MC[c * MC_STRIDE + tid]; }
  else if (tid < 64 + (KB + 1) * KB) Vtop[tid - 64] = MC[c * MC_STRIDE + tid];
  else if (tid < 64 + 2 * (KB + 1) * KB) Wtop[tid - 64 - (KB + 1) * KB] = MC[c * MC_STRIDE + tid];
  // rows of the tile (coalesced: 64 consecutive rows per column q)
  Ysh[rl * (KB + 1) + q] = Yx[c * KB * (int64_t)Np + PIX(q, r)];
  Vsh[rl * (KB + 1) + q] = Vprev[c * KB * (int64_t)Np + PIX(q, r)];
  // the tile's piece of the columns to update: loaded now, used after the barriers
  cplx bcol[2];
#pragma unroll
  for (int u = 0; u < 2; ++u) {
    const int cc = q + 8 * u, col = jprev + cc;
    bcol[u] = (cc < ncol && r >= col && r < N) ? B[r + (int64_t)col * N] : mkc(0.0, 0.0);
  }
  __syncthreads();
  cplx w = mkc(0.0, 0.0);
#pragma unroll
  for (int k1 = 0; k1 < KB; ++k1) { cfma(w, Ysh[rl * (KB + 1) + k1], Ts[k1 * KB + q]); cfms(w, Vsh[rl * (KB + 1) + k1], Cs[k1 * KB + q]); }
  Wsh[rl * (KB + 1) + q] = w;
  Wx[c * KB * (int64_t)Np + PIX(q, r)] = (r >= j2 && r < N) ? w : mkc(0.0, 0.0);
  __syncthreads();
#pragma unroll
  for (int u = 0; u < 2; ++u) {
    const int cc = q + 8 * u, col = jprev + cc;
    if (cc < ncol && r >= col && r < N) {
      cplx acc = bcol[u];
#pragma unroll
      for (int k1 = 0; k1 < KB; ++k1) {
        cfms(acc, Wsh[rl * (KB + 1) + k1], cconj(Vtop[cc * KB + k1]));
        cfms(acc, Vsh[rl * (KB + 1) + k1], cconj(Wtop[cc * KB + k1]));
      }
      if (r == col) acc.y = 0.0;
      B[r + (int64_t)col * N] = acc;
    }
  }
}

// QR step of panel p, one CTA per matrix: Householder QR of the columns p KB .. p KB + KB - 1 below row
// j2 = (p + 1) KB (thread t owns the rows j2 + t + s PT): reflectors stored in place (R on and above the
// sub-band diagonal), explicit V (unit heads, zeros above) for k_fused, tau, T; one block reduction per column.
// The panel stays on chip: row slot 0 of every thread in registers, the slots s >= 1 in shared memory
// ([slot][column][thread]: conflict free).
template <int RPT>
__global__ void __launch_bounds__(PT, 1) k_panel(cplx* __restrict__ Bw, cplx* __restrict__ Vnew, cplx* __restrict__ Vprev,
                                                 cplx* __restrict__ Wx, cplx* __restrict__ T1, cplx* __restrict__ tau1,
                                                 int N, int Np, int p) {
  extern __shared__ __align__(16) cplx psm[];   // panel slots 1 .. RPT-1
  __shared__ cplx Tn[KB * KB];
  __shared__ cplx red[(PT / 32) * KB], res[2][KB], head[2][KB];
  const int64_t c = blockIdx.x;
  const int tid = threadIdx.x;
  cplx* __restrict__ B = Bw + c * (int64_t)N * N;
  cplx* __restrict__ Vn = Vnew + c * KB * (int64_t)Np;
  cplx* __restrict__ Vp = Vprev + c * KB * (int64_t)Np;
  cplx* __restrict__ W = Wx + c * KB * (int64_t)Np;
  const int jprev = p * KB, j2 = jprev + KB;
  cplx a0[KB];
#define PA(s, q) psm[(((s) - 1) * KB + (q)) * PT + tid]
#pragma unroll
  for (int s = 0; s < RPT; ++s) {
    const int r = j2 + tid + s * PT;
#pragma unroll
    for (int cc = 0; cc < KB; ++cc) {
      const cplx t = (r < N) ? B[r + (int64_t)(jprev + cc) * N] : mkc(0.0, 0.0);
      if (s == 0) a0[cc] = t; else PA(s, cc) = t;
    }
  }
  if (tid < 64) Tn[tid] = mkc(0.0, 0.0);

  // ---- Householder QR (local row lr = r - j2; the thread's slot s holds lr = tid + s PT)
  const int lr0 = tid;
#pragma unroll 1
  for (int cc = 0; cc < KB; ++cc) {
    const int hb = cc & 1;
    if (tid == cc) {
#pragma unroll
      for (int q = 0; q < KB; ++q) head[hb][q] = a0[q];
    }
    cplx part[KB];
#pragma unroll
    for (int q = 0; q < KB; ++q) part[q] = mkc(0.0, 0.0);
#pragma unroll
    for (int s = 0; s < RPT; ++s) {
      const int lr = lr0 + s * PT;
      if (lr > cc && j2 + lr < N) {
        cplx row[KB];
#pragma unroll
        for (int q = 0; q < KB; ++q) row[q] = (s == 0) ? a0[q] : PA(s, q);
        cplx ac = row[0];
#pragma unroll
        for (int q = 1; q < KB; ++q) if (q == cc) ac = row[q];
#pragma unroll
        for (int q = 0; q < KB; ++q) {
          if (q >= cc) cfmac(part[q], ac, row[q]);   // conj(a_cc) a_q
          else cfmac(part[q], row[q], ac);           // conj(v_q) a_cc
        }
      }
    }
    block_sum8(part, red, res[hb]);
    const cplx alpha = head[hb][cc];
    const double xn2 = res[hb][cc].x;
    cplx tau, scale, betac;
    if (xn2 == 0.0) {
      tau = mkc(0.0, 0.0); scale = mkc(0.0, 0.0); betac = alpha;
    } else {
      double beta;
      larfg_scalars(alpha, xn2, beta, tau, scale);
      betac = mkc(beta, 0.0);
    }
    // f[q] = conj(tau) (head[q] + conj(scale) g[q]),  q > cc
    cplx f[KB];
#pragma unroll
    for (int q = 0; q < KB; ++q) {
      f[q] = mkc(0.0, 0.0);
      if (q > cc) {
        cplx t = head[hb][q];
        cfmac(t, scale, res[hb][q]);
        f[q] = cmulc(tau, t);
      }
    }
#pragma unroll
    for (int s = 0; s < RPT; ++s) {
      const int lr = lr0 + s * PT;
      if (lr >= cc && j2 + lr < N) {
        cplx row[KB];
#pragma unroll
        for (int q = 0; q < KB; ++q) row[q] = (s == 0) ? a0[q] : PA(s, q);
        cplx ac = row[0];
#pragma unroll
        for (int q = 1; q < KB; ++q) if (q == cc) ac = row[q];
        const cplx vv = (lr > cc) ? cmul(ac, scale) : mkc(1.0, 0.0);
#pragma unroll
        for (int q = 0; q < KB; ++q) {
          if (q > cc) cfms(row[q], f[q], vv);
          else if (q == cc) row[q] = (lr > cc) ? vv : betac;
        }
#pragma unroll
        for (int q = 0; q < KB; ++q) { if (s == 0) a0[q] = row[q]; else PA(s, q) = row[q]; }
      }
    }
    if (tid == 0) {
      // column cc of T:  T[0:cc, cc] = -tau T[0:cc, 0:cc] z,  z[q] = V_q^H v_cc = conj(v_q[cc]) + scale sum_{lr>cc} conj(v_q) a_cc
      cplx z[KB];
#pragma unroll
      for (int q = 0; q < KB; ++q) {
        z[q] = mkc(0.0, 0.0);
        if (q < cc) { z[q] = cconj(head[hb][q]); cfma(z[q], scale, res[hb][q]); }
      }
      for (int q = 0; q < cc; ++q) {
        cplx t = mkc(0.0, 0.0);
        for (int q2 = q; q2 < cc; ++q2) cfma(t, Tn[q * KB + q2], z[q2]);
        Tn[q * KB + cc] = cmul(mkc(-tau.x, -tau.y), t);
      }
      Tn[cc * KB + cc] = tau;
      tau1[c * N + jprev + cc] = tau;
    }
  }
  __syncthreads();
  if (tid < 64) T1[c * 64 + tid] = Tn[tid];
  // ---- write the panel back: R / v in place, explicit V for k_fused
#pragma unroll
  for (int s = 0; s < RPT; ++s) {
    const int lr = lr0 + s * PT;
    const int r = j2 + lr;
    if (lr >= 0 && r < N) {
#pragma unroll
      for (int cc = 0; cc < KB; ++cc) {
        const cplx t = (s == 0) ? a0[cc] : PA(s, cc);
        B[r + (int64_t)(jprev + cc) * N] = t;
        Vn[PIX(cc, r)] = (lr > cc) ? t : (lr == cc ? mkc(1.0, 0.0) : mkc(0.0, 0.0));
      }
    }
  }
  if (tid < KB) {
    const int r = jprev + tid;
    if (r < Np) {
#pragma unroll
      for (int q = 0; q < KB; ++q) {
        Vn[PIX(q, r)] = mkc(0.0, 0.0);
        Vp[PIX(q, r)] = mkc(0.0, 0.0);
        W[PIX(q, r)] = mkc(0.0, 0.0);
      }
    }
  }
#undef PA
}

// ------------------------------------------------------------------------------------------
// The streaming kernel of stage 1.  Work item = (matrix c, block column J); the CTA walks down the tiles
// (I, J), I = J .. nT-1.  Per tile:
//   1  A_IJ -= W_I V_J^H + V_I W_J^H          previous panel (K = 2 KB), accumulators start from the tile
//   2  A_IJ goes back to shared memory and from there to HBM (bulk store)
//   3  Y_I += A_IJ V+_J                        the accumulators are the A operand (no shared-memory round trip)
//   4  Y_J += A_IJ^H V+_I   (I != J)           the tile in shared memory is the B operand of (V+_I)^H A_IJ
// A producer warp runs two tiles ahead (TMA bulk copies, mbarrier complete_tx), issues the bulk stores and
// fetches items from a global counter (longest block columns first); 8 consumer warps, warp w owns the rows
// 8w .. 8w+7 of the tile in steps 1-3 and the columns 8w .. 8w+7 in step 4.  Row parts go to P[c][J][r][.]
// (k_panel adds the block columns: no atomics), the column part stays in registers over the whole item.
constexpr int FUSED_THREADS = 288;
constexpr size_t F_OFF_VPI = (size_t)2 * TS * LDT * sizeof(cplx);
constexpr size_t F_OFF_J = F_OFF_VPI + (size_t)2 * KB * LDR * sizeof(cplx);
constexpr size_t F_OFF_BAR = F_OFF_J + (size_t)2 * 3 * KB * LDR * sizeof(cplx);
constexpr size_t FUSED_SMEM = F_OFF_BAR + 6 * sizeof(unsigned long long) + 4 * sizeof(int4) + 16;

__device__ __forceinline__ void bulk_s2g(void* gdst, const void* ssrc, uint32_t bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(gdst), "r"(smem_u32(ssrc)), "r"(bytes)
               : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait0() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }

__global__ void __launch_bounds__(FUSED_THREADS, 1)
k_fused(cplx* __restrict__ Bw, const cplx* __restrict__ Vnew, const cplx* __restrict__ Vprev,
        const cplx* __restrict__ Wx, cplx* __restrict__ P, cplx* __restrict__ Zc, int N, int Np, int nT, int J0,
        int cnt, int has_upd, int* __restrict__ counter, int total) {
  extern __shared__ __align__(128) unsigned char fsm[];
  cplx* At = (cplx*)fsm;                                   // [2][TS cols][LDT]
  cplx* VpI = (cplx*)(fsm + F_OFF_VPI);                    // [2][KB][LDR]
  cplx* Jp = (cplx*)(fsm + F_OFF_J);                       // [2][3][KB][LDR]: V- (prev), W- (prev), V+ (new) rows of J
  unsigned long long* full = (unsigned long long*)(fsm + F_OFF_BAR);
  unsigned long long* empty = full + 2;
  unsigned long long* stready = full + 4;
  volatile int4* desc = (volatile int4*)(full + 6);        // ring of 4 tile descriptors {c, J, I, flags}
  volatile int* published = (volatile int*)(desc + 4);
  const int tid = threadIdx.x;
  if (tid == 0) {
    for (int s = 0; s < 2; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 8); mbar_init(&stready[s], 1); }
    *published = 0;
    mbar_fence_init();
  }
  // stale tile data is multiplied by exact zeros of the panels (rows / columns beyond N): keep it finite
  for (int idx = tid; idx < 2 * TS * LDT; idx += FUSED_THREADS) At[idx] = mkc(0.0, 0.0);
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  __syncthreads();
  constexpr uint32_t PANEL_BYTES = KB * TS * sizeof(cplx);   // KB column segments of TS rows

  if (tid >= 256) {
    // ------------------------------- producer warp
    const int lane = tid - 256;
    int gt = 0, itemseq = 0;
    int next = 0;
    if (lane == 0) next = atomicAdd(counter, 1);
    int pc = 0, pJ = 0, pI = 0;          // previous tile (its store is issued one tile later)
    bool have_prev = false;
    for (;;) {
      const int item = __shfl_sync(0xffffffffu, next, 0);
      if (lane == 0 && item < total) next = atomicAdd(counter, 1);
      if (item >= total) break;
      const int jj = item / cnt;
      const int c = item - jj * cnt;
      const int J = J0 + jj;
      for (int I = J; I < nT; ++I, ++gt) {
        const int s = gt & 1;
        if (gt >= 2) { mbar_wait(&empty[s], ((gt >> 1) - 1) & 1); bulk_wait_read0(); }
        const int r0 = I * TS, c0 = J * TS;
        const int nr = (N - r0 < TS) ? N - r0 : TS;
        const int nc = (N - c0 < TS) ? N - c0 : TS;
        const bool first = (I == J);
        if (lane == 0) {
          int4 d; d.x = c; d.y = J; d.z = I; d.w = (first ? 1 : 0) | (I == nT - 1 ? 2 : 0);
          desc[gt & 3].x = d.x; desc[gt & 3].y = d.y; desc[gt & 3].z = d.z; desc[gt & 3].w = d.w;
          __threadfence_block();
          *published = gt + 1;
          mbar_expect_tx(&full[s], (uint32_t)nc * nr * sizeof(cplx) + PANEL_BYTES + (first ? 3 * PANEL_BYTES : 0));
        }
        __syncwarp();
        const cplx* B = Bw + (int64_t)c * N * N;
        cplx* at = At + (size_t)s * TS * LDT;
        for (int col = lane; col < nc; col += 32)
          tma_bulk_g2s(at + col * LDT, B + r0 + (int64_t)(c0 + col) * N, (uint32_t)nr * sizeof(cplx), &full[s]);
        if (lane < KB)
          tma_bulk_g2s(VpI + ((size_t)s * KB + lane) * LDR, Vnew + (int64_t)c * KB * Np + PIX(lane, r0), TS * sizeof(cplx), &full[s]);
        if (first && lane >= KB) {
          const int arr = (lane - KB) / KB, qq = (lane - KB) % KB;
          const cplx* src = (arr == 0 ? Vprev : (arr == 1 ? Wx : Vnew)) + (int64_t)c * KB * Np + PIX(qq, c0);
          tma_bulk_g2s(Jp + (((size_t)(itemseq & 1) * 3 + arr) * KB + qq) * LDR, src, TS * sizeof(cplx), &full[s]);
        }
        // the updated previous tile goes back to HBM as soon as the consumers have written it to shared memory
        if (has_upd && have_prev) {
          const int ps = (gt - 1) & 1;
          mbar_wait(&stready[ps], ((gt - 1) >> 1) & 1);
          const int pr0 = pI * TS, pc0 = pJ * TS;
          const int pnr = (N - pr0 < TS) ? N - pr0 : TS;
          const int pnc = (N - pc0 < TS) ? N - pc0 : TS;
          cplx* Bp = Bw + (int64_t)pc * N * N;
          const cplx* pat = At + (size_t)ps * TS * LDT;
          for (int col = lane; col < pnc; col += 32)
            bulk_s2g(Bp + pr0 + (int64_t)(pc0 + col) * N, pat + col * LDT, (uint32_t)pnr * sizeof(cplx));
          bulk_commit();
        }
        pc = c; pJ = J; pI = I; have_prev = true;
      }
      ++itemseq;
    }
    if (has_upd && have_prev) {
      const int ps = (gt - 1) & 1;
      mbar_wait(&stready[ps], ((gt - 1) >> 1) & 1);
      const int pr0 = pI * TS, pc0 = pJ * TS;
      const int pnr = (N - pr0 < TS) ? N - pr0 : TS;
      const int pnc = (N - pc0 < TS) ? N - pc0 : TS;
      cplx* Bp = Bw + (int64_t)pc * N * N;
      const cplx* pat = At + (size_t)ps * TS * LDT;
      for (int col = lane; col < pnc; col += 32)
        bulk_s2g(Bp + pr0 + (int64_t)(pc0 + col) * N, pat + col * LDT, (uint32_t)pnr * sizeof(cplx));
      bulk_commit();
    }
    // stop mark
    {
      const int s = gt & 1;
      if (gt >= 2) mbar_wait(&empty[s], ((gt >> 1) - 1) & 1);
      if (lane == 0) {
        desc[gt & 3].x = -1;
        __threadfence_block();
        *published = gt + 1;
        mbar_arrive(&full[s]);
      }
    }
    bulk_wait0();
    return;
  }

  // ------------------------------- consumers
  const int lane = tid & 31, w = tid >> 5, g = lane >> 2, q = lane & 3;
  // column part of the item in 3-product form (two chains each)
  double zs1[2][2] = {{0.0, 0.0}, {0.0, 0.0}}, zs2[2][2] = {{0.0, 0.0}, {0.0, 0.0}}, zs3[2][2] = {{0.0, 0.0}, {0.0, 0.0}};
  int jb = 1;
  cplx Lw[2], Lv[2];          // fragments of [W- V-] rows of the tile, k = 2q, 2q+1
  int Lfor = -1;              // tile number these fragments were fetched for
  for (int gt = 0;; ++gt) {
    const int s = gt & 1;
    mbar_wait(&full[s], (gt >> 1) & 1);
    const int c = desc[gt & 3].x;
    if (c < 0) break;
    const int J = desc[gt & 3].y, I = desc[gt & 3].z, fl = desc[gt & 3].w;
    if (fl & 1) jb ^= 1;
    const cplx* at = At + (size_t)s * TS * LDT;
    const cplx* vpi = VpI + (size_t)s * KB * LDR;
    const cplx* VmJ = Jp + ((size_t)jb * 3 + 0) * KB * LDR;
    const cplx* WmJ = Jp + ((size_t)jb * 3 + 1) * KB * LDR;
    const cplx* VpJ = Jp + ((size_t)jb * 3 + 2) * KB * LDR;
    const int rI = I * TS + 8 * w + g;    // < Np always
    cplx lw0, lw1, lv0, lv1;
    if (has_upd) {
      if (Lfor != gt) {
        const cplx* wr = Wx + (int64_t)c * KB * Np + PIX(2 * q, rI);
        const cplx* vr = Vprev + (int64_t)c * KB * Np + PIX(2 * q, rI);
        Lw[0] = wr[0]; Lw[1] = wr[Np]; Lv[0] = vr[0]; Lv[1] = vr[Np];
      }
      lw0 = Lw[0]; lw1 = Lw[1]; lv0 = Lv[0]; lv1 = Lv[1];
    }
    // accumulators <- tile: thread holds A[8w+g][8nb + 2q + j]
    double ar[8][2], ai[8][2];
#pragma unroll
    for (int nb = 0; nb < 8; ++nb)
#pragma unroll
      for (int j = 0; j < 2; ++j) {
        const cplx t = at[(8 * nb + 2 * q + j) * LDT + 8 * w + g];
        ar[nb][j] = t.x; ai[nb][j] = t.y;
      }
    if (has_upd) {
      // step 1: C -= L R^H, L = [W_I V_I], R = [V_J W_J]:  Re -= Lr Rr + Li Ri,  Im -= Li Rr - Lr Ri
      const double l_r[4] = {lw0.x, lw1.x, lv0.x, lv1.x};
      const double l_i[4] = {lw0.y, lw1.y, lv0.y, lv1.y};
#pragma unroll
      for (int nb = 0; nb < 8; ++nb) {
#pragma unroll
        for (int ks = 0; ks < 4; ++ks) {
          const cplx rj = (ks < 2 ? VmJ : WmJ)[(2 * q + (ks & 1)) * LDR + 8 * nb + g];
          dmma(ar[nb][0], ar[nb][1], -l_r[ks], rj.x);
          dmma(ar[nb][0], ar[nb][1], -l_i[ks], rj.y);
          dmma(ai[nb][0], ai[nb][1], -l_i[ks], rj.x);
          dmma(ai[nb][0], ai[nb][1], l_r[ks], rj.y);
        }
      }
      // step 2: back to shared memory (same positions); the bulk store by the producer follows the barrier below
      cplx* atw = At + (size_t)s * TS * LDT;
#pragma unroll
      for (int nb = 0; nb < 8; ++nb)
#pragma unroll
        for (int j = 0; j < 2; ++j) atw[(8 * nb + 2 * q + j) * LDT + 8 * w + g] = mkc(ar[nb][j], ai[nb][j]);
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      // fragments of the next tile (the producer announced it when this tile started: no race by now)
      if (*published > gt + 1) {
        const int nc2 = desc[(gt + 1) & 3].x, nI = desc[(gt + 1) & 3].z;
        if (nc2 >= 0) {
          const int nr2 = nI * TS + 8 * w + g;
          const cplx* wr = Wx + (int64_t)nc2 * KB * Np + PIX(2 * q, nr2);
          const cplx* vr = Vprev + (int64_t)nc2 * KB * Np + PIX(2 * q, nr2);
          Lw[0] = wr[0]; Lw[1] = wr[Np]; Lv[0] = vr[0]; Lv[1] = vr[Np];
          Lfor = gt + 1;
        }
      }
    }
    // step 3: Y_I[8w+g][n] += sum_col A[.][col] V+_J[col][n]; k index q <-> column 8nb + 2q + j.  Three real
    // products per complex one (Karatsuba): P1 = ar br, P2 = ai bi, P3 = (ar + ai)(br + bi); Re = P1 - P2,
    // Im = P3 - P1 - P2 -- the operand sums cost one DADD each, a quarter of the DMMAs is saved.
    {
      double y1[2][2] = {{0.0, 0.0}, {0.0, 0.0}}, y2[2][2] = {{0.0, 0.0}, {0.0, 0.0}}, y3[2][2] = {{0.0, 0.0}, {0.0, 0.0}};
#pragma unroll
      for (int nb = 0; nb < 8; ++nb)
#pragma unroll
        for (int j = 0; j < 2; ++j) {
          const cplx b = VpJ[g * LDR + 8 * nb + 2 * q + j];
          const int ch = nb & 1;
          dmma(y1[ch][0], y1[ch][1], ar[nb][j], b.x);
          dmma(y2[ch][0], y2[ch][1], ai[nb][j], b.y);
          dmma(y3[ch][0], y3[ch][1], ar[nb][j] + ai[nb][j], b.x + b.y);
        }
      cplx* pr = P + ((int64_t)c * nT + J) * KB * Np + PIX(2 * q, rI);
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const double p1 = y1[0][e] + y1[1][e], p2 = y2[0][e] + y2[1][e], p3 = y3[0][e] + y3[1][e];
        pr[(int64_t)e * Np] = mkc(p1 - p2, p3 - p1 - p2);
      }
    }
    if (has_upd) {
      // every warp's part of the updated tile is in shared memory: release the bulk store, start step 4
      asm volatile("bar.sync 1, 256;" ::: "memory");
      if (tid == 0) mbar_arrive(&stready[s]);
    }
    // step 4: Z[m][col] += sum_row conj(V+_I[row][m]) A[row][col], col = 8w + n;  Y_J[col][m] = conj(Z[m][col]).
    // Karatsuba again: S1 = sum vr br, S2 = sum vi bi, S3 = sum (vr - vi)(br + bi); Re Z = S1 + S2, Im Z = S3 - S1 + S2
    if (I != J) {
#pragma unroll
      for (int blk = 0; blk < 8; ++blk)
#pragma unroll
        for (int j = 0; j < 2; ++j) {
          const int row = 8 * blk + 2 * q + j;
          const cplx v = vpi[g * LDR + row];
          const cplx b = at[(8 * w + g) * LDT + row];
          const int ch = blk & 1;
          dmma(zs1[ch][0], zs1[ch][1], v.x, b.x);
          dmma(zs2[ch][0], zs2[ch][1], v.y, b.y);
          dmma(zs3[ch][0], zs3[ch][1], v.x - v.y, b.x + b.y);
        }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(&empty[s]);
    if (fl & 2) {
      // end of the item: column part of block column J
#pragma unroll
      for (int j = 0; j < 2; ++j) {
        const int col = J * TS + 8 * w + 2 * q + j;
        const double s1 = zs1[0][j] + zs1[1][j], s2 = zs2[0][j] + zs2[1][j], s3 = zs3[0][j] + zs3[1][j];
        Zc[(int64_t)c * KB * Np + PIX(g, col)] = mkc(s1 + s2, -((s3 - s1) + s2));
        zs1[0][j] = zs1[1][j] = zs2[0][j] = zs2[1][j] = zs3[0][j] = zs3[1][j] = 0.0;
      }
    }
  }
}

// ------------------------------------------------------------------------------------------
// Compact band storage for the chase: AB[c][j][d] = A[j + d][j], d = 0 .. 2 KB - 1 (the fill of the
// bulges reaches 2 KB - 1 below the diagonal), zero where nothing is stored.
__global__ void k_band_extract(const cplx* __restrict__ Bw, cplx* __restrict__ AB, int N) {
  const int64_t c = blockIdx.y;
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= N * LDAB) return;
  const int j = idx / LDAB, d = idx % LDAB;
  cplx v = mkc(0.0, 0.0);
  if (d <= KB && j + d < N) v = Bw[c * (int64_t)N * N + (j + d) + (int64_t)j * N];
  if (d == 0) v.y = 0.0;
  AB[c * (int64_t)N * LDAB + idx] = v;
}

// Bulge chasing, one CTA per matrix.  The G sweeps i0 .. i0 + G - 1 of a "train" run two chase steps apart
// (sweep i0 + s does step k = t - 2s at time t), so everything the train touches at time t lies in a window of
// 15 G + 16 columns of the band, which is kept in a ring buffer in shared memory: per time step 8 columns enter at
// the front (cp.async, fetched three steps ahead) and 8 leave at the back.  Step (i, k), reflector on the rows
// st = i + 1 + k KB ..:
//   k > 0: E = A[R_k, R_{k-1}] <- E H_{k-1};  H_k from E[:, 0];  E <- H_k^H E
//   k = 0: H_0 from A[R_0, i]
//   D = A[R_k, R_k] <- H_k^H D H_k
// The reflector (tau in the head slot) is stored in the upper triangle of the work matrix: V2(i, rho) at
// Bw[i + rho N], rho = row the entry acts on.
constexpr int CH_RING = 256;     // columns of the ring buffer (>= 15 G + 16 + 8 * 3)

// FOUR sweeps per warp: a group of 8 lanes owns one chase step, lane r its row r of the two KB x KB blocks (E: 8
// entries, D: the full Hermitian row, 8 entries).  Row-wise products are lane-local, the column-wise ones (v^H E,
// v^H p) are 8-lane butterflies; the vectors every lane needs in full (v, w, v^H E) go through a few bytes of
// shared memory per group.  (A first version with one step per WARP, 2 of the 64 block entries per lane, was
// issue bound at ~450 instructions per step -- ncu, profiles/r02_chase_ncu_details.md: 56 vs 41 ms per 300
// matrices of N = 1600.)  G = 4 x warps = 12 sweeps in flight, three CTAs per SM.
constexpr int CH4_WMAX = 3;      // warps per CTA: 12 sweeps in flight, window 15 * 12 + 25 <= CH_RING
__global__ void __launch_bounds__(CH4_WMAX * 32) k_chase4(cplx* __restrict__ ABw, cplx* __restrict__ Bw, double* __restrict__ dd,
                                                         double* __restrict__ ee, int N) {
  static_assert(KB == 8, "lane mapping written for KB = 8");
  extern __shared__ __align__(16) cplx ring[];   // [CH_RING][LDAB], then the per-group vectors
  const int64_t c = blockIdx.x;
  cplx* __restrict__ abg = ABw + c * (int64_t)N * LDAB;
  cplx* __restrict__ Bc = Bw + c * (int64_t)N * N;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, G = (blockDim.x >> 5) * 4;
  const int r = lane & 7, grp = lane >> 3, slot = warp * 4 + grp;
  cplx* vsm = ring + CH_RING * LDAB + slot * 3 * KB;   // v of the current / previous step
  cplx* zsm = vsm + KB;                                 // v^H E
  cplx* wsm = vsm + 2 * KB;                             // w of the two-sided update
  for (int idx = tid; idx < (int)(blockDim.x >> 5) * 4 * 3 * KB; idx += blockDim.x) ring[CH_RING * LDAB + idx] = mkc(0.0, 0.0);
  __syncthreads();
#define RG(col, d) ring[((col) & (CH_RING - 1)) * LDAB + (d)]
  auto load_cols = [&](int c0, int c1) {
    if (c1 > N) c1 = N;
    for (int idx = tid; idx < (c1 - c0) * LDAB; idx += blockDim.x) {
      const int col = c0 + idx / LDAB, d = idx % LDAB;
      const uint32_t dst = smem_u32(&RG(col, d));
      asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(dst), "l"(abg + (int64_t)col * LDAB + d) : "memory");
    }
  };
  auto store_cols = [&](int c0, int c1) {
    if (c1 > N) c1 = N;
    for (int idx = tid; idx < (c1 - c0) * LDAB; idx += blockDim.x) {
      const int col = c0 + idx / LDAB, d = idx % LDAB;
      abg[(int64_t)col * LDAB + d] = RG(col, d);
    }
  };
  for (int i0 = 0; i0 < N - 1; i0 += G) {
    const int i = i0 + slot;
    const int T = (N - 1 - i0 + KB - 1) / KB + 2 * (G - 1);
    int back = i0;
    // columns enter three time steps before they are needed (an L2 round trip is longer than a step)
    int front = (i0 + 9 + 16 < N) ? i0 + 9 + 16 : N;
    load_cols(i0, front);
    asm volatile("cp.async.commit_group;\n" ::: "memory");
    asm volatile("cp.async.commit_group;\n" ::: "memory");
    asm volatile("cp.async.commit_group;\n" ::: "memory");
    cplx tauprev = mkc(0.0, 0.0);
    for (int t = 0; t < T; ++t) {
      asm volatile("cp.async.wait_group 2;\n" ::: "memory");
      __syncthreads();
      {
        const int nf = (i0 + 8 * (t + 3) + 9 < N) ? i0 + 8 * (t + 3) + 9 : N;
        if (nf > front) { load_cols(front, nf); front = nf; }
        asm volatile("cp.async.commit_group;\n" ::: "memory");
        int nb = i0 + G + 8 * (t - 2 * (G - 1)) - 16;
        if (nb > front) nb = front;
        if (nb > back) { store_cols(back, nb); back = nb; }
      }
      const int k = t - 2 * slot;
      const int st = i + 1 + k * KB;
      const bool act = (i < N - 1) && (k >= 0) && (st < N);
      // whole warp idle: nothing to do (uniform)
      if (!__any_sync(0xffffffffu, act)) continue;
      const int len = act ? ((N - st < KB) ? N - st : KB) : 0;
      const bool first = (k == 0);
      const bool rowok = r < len;
      // ---- loads: row r of E (k > 0) or the entry of column i (k = 0), and the full row r of D
      cplx e[KB], d[KB];
#pragma unroll
      for (int cc = 0; cc < KB; ++cc) {
        e[cc] = mkc(0.0, 0.0); d[cc] = mkc(0.0, 0.0);
        if (rowok && !first) e[cc] = RG(st - KB + cc, KB + r - cc);
        if (rowok && cc < len) {
          const bool lo = r >= cc;
          const int c2 = lo ? st + cc : st + r, o2 = lo ? r - cc : cc - r;
          cplx t2 = RG(c2, o2);
          if (!lo) t2.y = -t2.y;
          d[cc] = t2;
        }
      }
      if (rowok && first) e[0] = RG(i, 1 + r);
      // ---- E <- E H_{k-1}  (v of the previous step is still in vsm; tau = 0 for k = 0)
      {
        cplx wv = mkc(0.0, 0.0);
#pragma unroll
        for (int cc = 0; cc < KB; ++cc) cfma(wv, e[cc], vsm[cc]);
        const cplx tw = cmul(first ? mkc(0.0, 0.0) : tauprev, wv);
#pragma unroll
        for (int cc = 0; cc < KB; ++cc) cfms(e[cc], tw, cconj(vsm[cc]));
      }
      __syncwarp();
      // ---- reflector from column 0 of E
      const cplx x = e[0];
      const cplx alpha = shfl_c(x, lane & 24);
      double xn2 = (r >= 1 && rowok) ? cabs2(x) : 0.0;
      xn2 += __shfl_xor_sync(0xffffffffu, xn2, 1);
      xn2 += __shfl_xor_sync(0xffffffffu, xn2, 2);
      xn2 += __shfl_xor_sync(0xffffffffu, xn2, 4);
      double beta; cplx tau, scale;
      if (xn2 == 0.0 && alpha.y == 0.0) {
        beta = alpha.x; tau = mkc(0.0, 0.0); scale = mkc(0.0, 0.0);
      } else {
        larfg_scalars(alpha, xn2, beta, tau, scale);
      }
      const cplx v = (r == 0) ? mkc(1.0, 0.0) : (rowok ? cmul(x, scale) : mkc(0.0, 0.0));
      vsm[r] = v;
      if (act && rowok) Bc[i + (int64_t)(st + r) * N] = (r == 0) ? tau : v;
      if (act && first && r == 0) { ee[c * N + i] = beta; dd[c * N + i] = RG(i, 0).x; }
      // ---- E <- H^H E: z[cc] = sum_r conj(v_r) e_r[cc] by an 8-lane halving butterfly (lane r ends with z[r])
      {
        cplx pz[KB];
#pragma unroll
        for (int cc = 0; cc < KB; ++cc) pz[cc] = cmulc(v, e[cc]);
        const bool u4 = r & 4, u2 = r & 2, u1 = r & 1;
        cplx b4[4], b2[2], b1;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const cplx snd = u4 ? pz[j] : pz[j + 4], kp = u4 ? pz[j + 4] : pz[j];
          b4[j] = cadd(kp, shfl_xor_c(snd, 4));
        }
#pragma unroll
        for (int j = 0; j < 2; ++j) {
          const cplx snd = u2 ? b4[j] : b4[j + 2], kp = u2 ? b4[j + 2] : b4[j];
          b2[j] = cadd(kp, shfl_xor_c(snd, 2));
        }
        {
          const cplx snd = u1 ? b2[0] : b2[1], kp = u1 ? b2[1] : b2[0];
          b1 = cadd(kp, shfl_xor_c(snd, 1));
        }
        zsm[r] = b1;   // index (u4 ? 4 : 0) + (u2 ? 2 : 0) + (u1 ? 1 : 0) = r
      }
      __syncwarp();
      cplx vc[KB];
#pragma unroll
      for (int cc = 0; cc < KB; ++cc) vc[cc] = vsm[cc];
      {
        const cplx ctv = cmul(cconj(tau), v);
#pragma unroll
        for (int cc = 1; cc < KB; ++cc) cfms(e[cc], ctv, zsm[cc]);
        e[0] = (r == 0) ? mkc(beta, 0.0) : mkc(0.0, 0.0);
      }
      if (act && rowok) {
        if (first) RG(i, 1 + r) = e[0];
        else {
#pragma unroll
          for (int cc = 0; cc < KB; ++cc) RG(st - KB + cc, KB + r - cc) = e[cc];
        }
      }
      // ---- D <- H^H D H = D - w v^H - v w^H,  w = tau p - 1/2 |tau|^2 (v^H p) v,  p = D v
      {
        cplx pp = mkc(0.0, 0.0);
#pragma unroll
        for (int cc = 0; cc < KB; ++cc) cfma(pp, d[cc], vc[cc]);
        double al = v.x * pp.x + v.y * pp.y;
        al += __shfl_xor_sync(0xffffffffu, al, 1);
        al += __shfl_xor_sync(0xffffffffu, al, 2);
        al += __shfl_xor_sync(0xffffffffu, al, 4);
        cplx wv = cmul(tau, pp);
        const double hf = 0.5 * cabs2(tau) * al;
        wv.x -= hf * v.x; wv.y -= hf * v.y;
        wsm[r] = wv;
        __syncwarp();
#pragma unroll
        for (int cc = 0; cc < KB; ++cc) {
          cfms(d[cc], wv, cconj(vc[cc]));
          cfms(d[cc], v, cconj(wsm[cc]));
        }
        if (act && rowok) {
#pragma unroll
          for (int cc = 0; cc < KB; ++cc)
            if (cc <= r && cc < len) { cplx t2 = d[cc]; if (cc == r) t2.y = 0.0; RG(st + cc, r - cc) = t2; }
        }
      }
      tauprev = tau;
      __syncwarp();
    }
    asm volatile("cp.async.wait_group 0;\n" ::: "memory");
    __syncthreads();
    store_cols(back, front);
    __syncthreads();
  }
  if (tid == 0) { dd[c * N + N - 1] = abg[(int64_t)(N - 1) * LDAB].x; ee[c * N + N - 1] = 0.0; }
#undef RG
}

// ------------------------------------------------------------------------------------------
// X <- conj(Q2) X,  Q2 = prod_i prod_k H_{i,k}  (sweeps ascending; applied last sweep first).
// A thread owns one column of X (frames layout: column v of matrix c is contiguous) and a window of
// QWN = QG + KB rows in registers; a group of QG consecutive sweeps at chase step k acts on the matrix rows
// i0 + 1 + k KB + u, sweep i0 + s on the window rows u = s .. s + KB - 1, and the window slides down by KB
// rows per step.  QS such stages form a pipeline inside the CTA: stage j applies the sweeps
// I0 + (QS - 1 - j) QG .. and hands the KB rows it retires per step to stage j + 1 through shared memory,
// one step behind -- a pass over the column applies QS QG sweeps, so X is streamed N / (QS QG) times instead
// of N / QG times with the registers of a QG window.  Stage 0 takes its new rows from memory: they are
// fetched one step ahead with cp.async into the same kind of hand-over buffer, so no stage waits on HBM
// inside a step.  The reflectors of a step are staged in shared memory (cp.async, double buffered) and
// read as broadcasts.  (A variant with the real and imaginary parts of a column on two lanes -- half the
// registers, 15 instead of 12 warps -- executed 1.6x the instructions and was slower: 174 vs 142 ms.)
constexpr int QG = 16;
constexpr int QWN = QG + KB;
constexpr int QS = 3;
constexpr int Q2_TSG_MAX = 128;   // threads (columns) per stage (3 x 128 threads: 168 registers each)

__device__ __forceinline__ void cp_async16_z(void* sdst, const void* gsrc, bool pred) {
  const uint32_t d = smem_u32(sdst);
  const int sz = pred ? 16 : 0;
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(d), "l"(gsrc), "r"(sz) : "memory");
}

__global__ void __launch_bounds__(QS * Q2_TSG_MAX, 1) k_q2(const cplx* __restrict__ Bw, cplx* __restrict__ X, int N, int nv,
                                                          int tsg, int col0) {
  extern __shared__ __align__(16) cplx qsm[];
  cplx* vs = qsm;                                  // [2][QS][QG * KB]
  cplx* hand = qsm + 2 * QS * QG * KB;             // [2][QS][KB][tsg]: input rows of stage j (j = 0: from memory)
  const int64_t c = blockIdx.y;
  const cplx* __restrict__ Bc = Bw + c * (int64_t)N * N;
  const int j = threadIdx.x / tsg, tcol = threadIdx.x - j * tsg;
  const int v = col0 + blockIdx.x * tsg + tcol;
  const bool act = v < nv;
  cplx* __restrict__ x = X + (c * nv + (act ? v : 0)) * (int64_t)N;
  const int nsuper = (N - 1 + QS * QG - 1) / (QS * QG);
  auto stage_v = [&](int buf, int i0, int k) {
    // slot (u, jj): sweep s = u - jj, entry jj; matrix row rho = i0 + 1 + k KB + u, source Bc[(i0 + s) + rho N]
    cplx* dst = vs + ((size_t)buf * QS + j) * QG * KB;
    for (int idx = tcol; idx < (QG + KB - 1) * KB; idx += tsg) {
      const int u = idx / KB, jj = idx % KB;
      const int s = u - jj;
      if (s < 0 || s >= QG) continue;
      const int i = i0 + s, rho = i0 + 1 + k * KB + u;
      const bool ok = (i < N - 1) && (rho < N);
      cp_async16_z(&dst[s * KB + jj], ok ? (Bc + i + (int64_t)rho * N) : Bc, ok);
    }
  };
  // stage 0: the KB rows that enter the window at step k, rho = i0 + 1 + k KB + QG + u
  auto stage_x = [&](int buf, int i0, int k) {
    cplx* dst = hand + ((size_t)buf * QS) * KB * tsg;
#pragma unroll
    for (int u = 0; u < KB; ++u) {
      const int rho = i0 + 1 + k * KB + QG + u;
      const bool ok = act && rho < N;
      cp_async16_z(&dst[u * tsg + tcol], ok ? (x + rho) : x, ok);
    }
  };
  for (int sg = nsuper - 1; sg >= 0; --sg) {
    const int I0 = sg * QS * QG;
    const int i0 = I0 + (QS - 1 - j) * QG;                               // this stage's sweeps i0 .. i0 + QG - 1
    const int nk = (i0 + 1 < N) ? (N - i0 - 1 + KB - 1) / KB : 0;        // its chase steps
    const int nk_up = (i0 + QG + 1 < N) ? (N - i0 - QG - 1 + KB - 1) / KB : 0;   // those of the stage above
    const int NK = (N - I0 - 1 + KB - 1) / KB + QS - 1;                  // steps of the pipeline
    __syncthreads();   // the previous pass is complete (its stores are visible, its buffers free)
    cplx wnd[QWN];
#pragma unroll
    for (int u = 0; u < QG; ++u) {
      const int rho = i0 + 1 + u;
      wnd[u] = (act && rho < N) ? x[rho] : mkc(0.0, 0.0);
    }
#pragma unroll
    for (int u = QG; u < QWN; ++u) wnd[u] = mkc(0.0, 0.0);
    if (j == 0 && nk > 0) { stage_v(0, i0, 0); stage_x(1, i0, 0); }   // step kap reads hand[(kap - 1) & 1]
    asm volatile("cp.async.commit_group;\n" ::: "memory");
    for (int kap = 0; kap < NK; ++kap) {
      const int k = kap - j;
      asm volatile("cp.async.wait_group 0;\n" ::: "memory");
      __syncthreads();
      if (k + 1 >= 0 && k + 1 < nk) {
        stage_v((kap + 1) & 1, i0, k + 1);
        if (j == 0) stage_x(kap & 1, i0, k + 1);
      }
      asm volatile("cp.async.commit_group;\n" ::: "memory");
      if (k < 0 || k >= nk) continue;
      const int rho0 = i0 + 1 + k * KB;
      // the KB new rows of this step
      {
        const cplx* hb = hand + ((size_t)((kap - 1) & 1) * QS + j) * KB * tsg;
        const bool ok = (j == 0) || (k < nk_up);
#pragma unroll
        for (int u = 0; u < KB; ++u) wnd[QG + u] = ok ? hb[u * tsg + tcol] : mkc(0.0, 0.0);
      }
      const cplx* vb = vs + ((size_t)(kap & 1) * QS + j) * QG * KB;
#pragma unroll
      for (int s = QG - 1; s >= 0; --s) {
        // conj(H) = I - conj(tau) conj(v) v^T
        const cplx tau = vb[s * KB];
        cplx d0 = wnd[s], d1 = mkc(0.0, 0.0);
#pragma unroll
        for (int jj = 1; jj < KB; ++jj) {
          const cplx vj = vb[s * KB + jj];
          if (jj & 1) cfma(d1, vj, wnd[s + jj]); else cfma(d0, vj, wnd[s + jj]);
        }
        const cplx t = cmulc(tau, cadd(d0, d1));   // conj(tau) * dot
        wnd[s] = csub(wnd[s], t);
        // x_j -= t conj(v_j), all products with t.x first, then all with t.y: consecutive DFMAs share an operand
        // (register-file bandwidth, not the FP64 pipe, limits three-operand DFMA streams on this part)
        cplx vj[KB];
#pragma unroll
        for (int jj = 1; jj < KB; ++jj) vj[jj] = vb[s * KB + jj];
#pragma unroll
        for (int jj = 1; jj < KB; ++jj) {
          wnd[s + jj].x = fma(-t.x, vj[jj].x, wnd[s + jj].x);
          wnd[s + jj].y = fma(t.x, vj[jj].y, wnd[s + jj].y);
        }
#pragma unroll
        for (int jj = 1; jj < KB; ++jj) {
          wnd[s + jj].x = fma(-t.y, vj[jj].y, wnd[s + jj].x);
          wnd[s + jj].y = fma(-t.y, vj[jj].x, wnd[s + jj].y);
        }
      }
      // rows u < KB are final for this stage
      if (j == QS - 1) {
        if (act) {
#pragma unroll
          for (int u = 0; u < KB; ++u) if (rho0 + u < N) x[rho0 + u] = wnd[u];
        }
      } else {
        cplx* hb = hand + ((size_t)(kap & 1) * QS + j + 1) * KB * tsg;
#pragma unroll
        for (int u = 0; u < KB; ++u) hb[u * tsg + tcol] = wnd[u];
      }
#pragma unroll
      for (int u = 0; u < QG; ++u) wnd[u] = wnd[u + KB];
    }
    asm volatile("cp.async.wait_group 0;\n" ::: "memory");
  }
}

struct BandScratch {
  cplx *Vx0, *Vx1, *Wx, *Yx, *P, *Zc, *T1, *AB, *Mpart, *MC;
  int* counters;
  int* start;
};

size_t band_carve(char* base, int64_t cnt, int N, BandScratch* s) {
  size_t off = 0;
  auto take = [&](size_t bytes) { char* p = base ? base + off : nullptr; off += be_align256(bytes); return p; };
  const int nT = (N + TS - 1) / TS, Np = nT * TS;
  cplx* v0 = (cplx*)take((size_t)cnt * Np * KB * sizeof(cplx));
  cplx* v1 = (cplx*)take((size_t)cnt * Np * KB * sizeof(cplx));
  cplx* wx = (cplx*)take((size_t)cnt * Np * KB * sizeof(cplx));
  cplx* yx = (cplx*)take((size_t)cnt * Np * KB * sizeof(cplx));
  cplx* P = (cplx*)take((size_t)cnt * nT * Np * KB * sizeof(cplx));
  cplx* zc = (cplx*)take((size_t)cnt * Np * KB * sizeof(cplx));
  cplx* t1 = (cplx*)take((size_t)cnt * 64 * sizeof(cplx));
  cplx* ab = (cplx*)take((size_t)cnt * N * LDAB * sizeof(cplx));
  cplx* mp = (cplx*)take((size_t)cnt * nT * 64 * sizeof(cplx));
  cplx* mc = (cplx*)take((size_t)cnt * MC_STRIDE * sizeof(cplx));
  int* counters = (int*)take((size_t)(N / KB + 2) * sizeof(int));
  int* start = (int*)take((size_t)N * sizeof(int));
  if (s) *s = BandScratch{v0, v1, wx, yx, P, zc, t1, ab, mp, mc, counters, start};
  return off;
}

}  // namespace

size_t be_band_scratch_bytes(int64_t cnt, int N) { return band_carve(nullptr, cnt, N, nullptr); }

#define LAUNCH_CHECK() do { ctx->launches++; cudaError_t e__ = cudaGetLastError(); if (e__ != cudaSuccess) return (int)e__; } while (0)

// Stage 1 + stage 2 on the work copies Bw [cnt][N][N]: d, e of the real tridiagonal matrix, tau of the
// stage-1 reflectors (column j: head at row j + KB), stage-1 vectors below the band of Bw, stage-2
// reflectors in its upper triangle.
int be_band_reduce(be_ctx* ctx, cplx* Bw, int64_t cnt, int N, double* d, double* e, cplx* tau, void* scratch) {
  BE_TRY(be_band_stage1(ctx, Bw, cnt, N, tau, scratch));
  return be_band_stage2(ctx, Bw, cnt, N, d, e, scratch);
}

// Stage 1 (dense -> band) alone.  Everything it leaves behind is in Bw and tau, so it may be run on sub-ranges of
// a batch one after the other with the same scratch (carved for the sub-range) before ONE stage 2 over the batch.
int be_band_stage1(be_ctx* ctx, cplx* Bw, int64_t cnt, int N, cplx* tau, void* scratch) {
  if (N > BE_BAND_MAXN || N < 2 * KB) return BE_ERR_UNSUPPORTED;
  if (cnt > 0x7fffffffLL / 64) return BE_ERR_SHAPE;
  BandScratch s;
  band_carve((char*)scratch, cnt, N, &s);
  cudaStream_t st = ctx->stream;
  const int nT = (N + TS - 1) / TS, Np = nT * TS;
  // last panel with something to annihilate: rows below j2 = (p + 1) KB number N - j2 >= 2
  const int plast = (N - 2) / KB - 1;
  BE_CUDA(cudaMemsetAsync(s.Vx0, 0, (size_t)cnt * Np * KB * sizeof(cplx), st));
  BE_CUDA(cudaMemsetAsync(s.Vx1, 0, (size_t)cnt * Np * KB * sizeof(cplx), st));
  BE_CUDA(cudaMemsetAsync(s.Wx, 0, (size_t)cnt * Np * KB * sizeof(cplx), st));
  BE_CUDA(cudaMemsetAsync(s.counters, 0, (size_t)(N / KB + 2) * sizeof(int), st));
  BE_CUDA(cudaMemsetAsync(tau, 0, (size_t)cnt * N * sizeof(cplx), st));
  k_symdiag<<<dim3((unsigned)nT, (unsigned)cnt), 256, 0, st>>>(Bw, N);
  LAUNCH_CHECK();
  auto panel = [&](int p, int do_qr) -> int {
    cplx* vn = (p & 1) ? s.Vx1 : s.Vx0;
    cplx* vp = (p & 1) ? s.Vx0 : s.Vx1;
    be_prof_begin(ctx, PK_PANEL);
    const int n = N - p * KB;
    if (p > 0) {
      // two wide kernels: Y = sum of the partial products (+ the tiles' shares of V^H Y), then W and the update
      // of the next panel's columns
      const int J0 = (p * KB) / TS;
      k_ysum<<<dim3((unsigned)(nT - J0), (unsigned)cnt), 512, 0, st>>>(s.P, s.Zc, vp, s.Yx, s.Mpart, N, Np, nT, J0, p * KB);
      ctx->launches++;
      k_mc<<<(unsigned)cnt, 96, 0, st>>>(s.Yx, vp, s.Mpart, s.T1, s.MC, N, Np, nT, J0, p * KB);
      ctx->launches++;
      k_wupd<<<dim3((unsigned)(nT - J0), (unsigned)cnt), 512, 0, st>>>(Bw, s.Yx, vp, s.Wx, s.MC, s.T1, N, Np, J0,
                                                                      p * KB, do_qr ? KB : N - p * KB);
      ctx->launches++;
    }
    if (do_qr) {
      const int rpt = (N - (p + 1) * KB + PT - 1) / PT;
      const size_t psm = (size_t)(rpt - 1) * PT * KB * sizeof(cplx);
#define PANEL_CASE(R) case R: \
      BE_CUDA(cudaFuncSetAttribute(k_panel<R>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)psm)); \
      k_panel<R><<<(unsigned)cnt, PT, psm, st>>>(Bw, vn, vp, s.Wx, s.T1, tau, N, Np, p); break;
      switch (rpt) {
        PANEL_CASE(1) PANEL_CASE(2) PANEL_CASE(3) PANEL_CASE(4)
        default: return BE_ERR_UNSUPPORTED;
      }
#undef PANEL_CASE
    }
    be_prof_end(ctx, PK_PANEL, (double)cnt * n * 16.0 * (6.0 * KB + 0.5 * KB * ((n + TS - 1) / TS)), (double)cnt * n * 8.0 * 6 * KB * KB);
    LAUNCH_CHECK();
    return BE_OK;
  };
  BE_CUDA(cudaFuncSetAttribute(k_fused, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FUSED_SMEM));
  for (int p = 0; p <= plast; ++p) {
    BE_TRY(panel(p, 1));
    const int j2 = (p + 1) * KB;
    const int J0 = j2 / TS;
    const int64_t total = cnt * (int64_t)(nT - J0);
    const int64_t grid = total < (int64_t)ctx->sm_count ? total : (int64_t)ctx->sm_count;
    const cplx* vn = (p & 1) ? s.Vx1 : s.Vx0;
    const cplx* vp = (p & 1) ? s.Vx0 : s.Vx1;
    be_prof_begin(ctx, PK_FUSED);
    k_fused<<<(unsigned)grid, FUSED_THREADS, FUSED_SMEM, st>>>(Bw, vn, vp, s.Wx, s.P, s.Zc, N, Np, nT, J0, (int)cnt,
                                                               p > 0 ? 1 : 0, s.counters + p, (int)total);
    {
      // algorithmic traffic: the lower triangle of the trailing matrix read once and (p > 0) written once;
      // flops: rank-2KB update (8 n^2 KB on the lower half) + the two-sided product (8 n^2 KB)
      const double n = N - j2;
      be_prof_end(ctx, PK_FUSED, (double)cnt * 0.5 * n * (n + 1.0) * 16.0 * (p > 0 ? 2.0 : 1.0),
                  (double)cnt * 8.0 * n * n * KB * (p > 0 ? 2.0 : 1.0));
    }
    LAUNCH_CHECK();
  }
  return panel(plast + 1, 0);
}

// Stage 2 (band -> real tridiagonal by bulge chasing) for the whole batch.
int be_band_stage2(be_ctx* ctx, cplx* Bw, int64_t cnt, int N, double* d, double* e, void* scratch) {
  if (N > BE_BAND_MAXN || N < 2 * KB) return BE_ERR_UNSUPPORTED;
  BandScratch s;
  band_carve((char*)scratch, cnt, N, &s);
  cudaStream_t st = ctx->stream;
  k_band_extract<<<dim3((unsigned)((N * LDAB + 255) / 256), (unsigned)cnt), 256, 0, st>>>(Bw, s.AB, N);
  LAUNCH_CHECK();
  {
    const size_t sm4 = (size_t)(CH_RING * LDAB + CH4_WMAX * 4 * 3 * KB) * sizeof(cplx);
    BE_CUDA(cudaFuncSetAttribute(k_chase4, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm4));
    be_prof_begin(ctx, PK_CHASE);
    k_chase4<<<(unsigned)cnt, CH4_WMAX * 32, sm4, st>>>(s.AB, Bw, d, e, N);
    be_prof_end(ctx, PK_CHASE, (double)cnt * N * LDAB * 16.0, (double)cnt * 24.0 * N * (double)N * KB);
    LAUNCH_CHECK();
  }
  return BE_OK;
}

int be_band_q2(be_ctx* ctx, const cplx* Bw, cplx* X, int64_t cnt, int N, int nv) {
  if (nv <= 0) return BE_OK;
  // Columns per CTA: whole slabs of Q2_TSG_MAX columns, and the rest (nv = 800: 6 x 128 + 32) in a grid of its own
  // with narrow CTAs.  A CTA takes the same time whatever share of its warps is active (the 32 leftover columns in a
  // seventh 128-column slab cost a full slab: 135.6 ms per 148 matrices for nv = 800 .. 896 against 116.3 for 768),
  // but four 96-thread CTAs fit an SM where one 384-thread CTA does.
  const int nfull = nv / Q2_TSG_MAX;
  const int rem = nv - nfull * Q2_TSG_MAX;
  const int tsg_tail = (rem + 31) / 32 * 32;
  // The two grids run side by side (the narrow one on ctx->side_stream): a full-slab CTA owns the register file of
  // its SM, so the narrow CTAs take whole SMs too, four at a time, and the block scheduler packs the two kinds -- no
  // nearly empty last round of either grid (600 matrices, nv = 800: 24.3 rounds of full slabs + 1.01 of narrow CTAs).
  const bool both = nfull > 0 && rem > 0;
  if (both && !ctx->side_stream) {
    BE_CUDA(cudaStreamCreateWithFlags(&ctx->side_stream, cudaStreamNonBlocking));
    BE_CUDA(cudaEventCreateWithFlags(&ctx->ev_side[0], cudaEventDisableTiming));
    BE_CUDA(cudaEventCreateWithFlags(&ctx->ev_side[1], cudaEventDisableTiming));
  }
  BE_CUDA(cudaFuncSetAttribute(k_q2, cudaFuncAttributeMaxDynamicSharedMemorySize,
                               (int)(((size_t)2 * QS * QG * KB + (size_t)2 * QS * KB * Q2_TSG_MAX) * sizeof(cplx))));
  be_prof_begin(ctx, PK_Q2);
  if (both) {
    BE_CUDA(cudaEventRecord(ctx->ev_side[0], ctx->stream));
    BE_CUDA(cudaStreamWaitEvent(ctx->side_stream, ctx->ev_side[0], 0));
  }
  for (int part = 0; part < 2; ++part) {
    const int tsg = part == 0 ? Q2_TSG_MAX : tsg_tail;
    const int nslab = part == 0 ? nfull : (rem > 0 ? 1 : 0);
    if (nslab == 0) continue;
    const size_t smem = ((size_t)2 * QS * QG * KB + (size_t)2 * QS * KB * tsg) * sizeof(cplx);
    cudaStream_t qs = (part == 1 && both) ? ctx->side_stream : ctx->stream;
    k_q2<<<dim3((unsigned)nslab, (unsigned)cnt), QS * tsg, smem, qs>>>(Bw, X, N, nv, tsg, part == 0 ? 0 : nfull * Q2_TSG_MAX);
    if (part == 0 && rem > 0) LAUNCH_CHECK();
  }
  if (both) {
    BE_CUDA(cudaEventRecord(ctx->ev_side[1], ctx->side_stream));
    BE_CUDA(cudaStreamWaitEvent(ctx->stream, ctx->ev_side[1], 0));
  }
  be_prof_end(ctx, PK_Q2, (double)cnt * nv * N * 16.0 * ((N + QS * QG - 1) / (QS * QG)), (double)cnt * 8.0 * N * (double)N * nv);
  LAUNCH_CHECK();
  return BE_OK;
}
