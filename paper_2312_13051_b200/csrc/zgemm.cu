// Batched complex128 GEMM on the FP64 tensor cores of sm_100a.
//
// tcgen05.mma has no f64 kind, so the FP64 tensor path on Blackwell is the warp-level
// mma.sync.m8n8k4.f64 (SASS DMMA.8x8x4) fed from shared memory with the accumulators in registers.
// A complex product is four real DMMAs on split re/im operands: the interleaved complex128 input
// is de-interleaved while it is staged into shared memory, where transposition and conjugation
// are also applied (a sign flip), so every op(A), op(B) combination runs the same inner loop.
//
// Used for: the link overlaps M_j = U_j^dagger U_{j+1} (ring mode, closing phase Phi applied in
// the loader; Eq. 2), the ordered Wilson product, the rank-2k
// update of the blocked tridiagonalization, the compact-WY back-transform, U^dagger S U and the
// sector rotations of the spin-resolved loop.
//
// Two kernels share the tile shape (64 x 32 x 16 per CTA, 128 threads = 4 warps as 2 (M) x 2 (N), warp tile
// 32 x 16 = 4 x 2 DMMA blocks, three real DMMAs per complex block):
//   zgemm_async_kernel -- the default: interleaved operands brought in by 16-byte cp.async, 16-byte fragment
//                         loads, 152-160 registers, three CTAs per SM;
//   zgemm_kernel       -- register-staged loader that de-interleaves re/im (and applies the closing phase
//                         Phi) on the way into shared memory: the closing-phase link GEMM, the chunk pipeline
//                         and BE_GEMM_ASYNC=0.
#include "be_common.cuh"

namespace {

constexpr bool M3 = true;   // 3-multiplication complex product (see the main loop)
// 3M keeps three accumulator sets (~190 registers): 64 x 32 tiles on 128 threads, so that two CTAs still
// share an SM and one CTA's epilogue overlaps the other's main loop
constexpr int TM = 64, TN = M3 ? 32 : 64, TK = 16, LDS = 68;  // LDS % 16 == 4: conflict-free fragment loads
constexpr int NTHREADS = M3 ? 128 : 256;
constexpr int QA = TM * TK / NTHREADS, QB = TN * TK / NTHREADS;   // staged elements per thread
constexpr int LDK = 20;                              // k-contiguous operands: [mn][k], LDK % 16 == 4
constexpr int SM_PLANE = TM * LDK;                   // doubles per A plane (>= TK * LDS)
constexpr int LDSB = TN + 4;                         // B staged [k][n]: LDSB % 16 == 4 as well
constexpr int SM_PLANEB = TN * LDK > TK * LDSB ? TN * LDK : TK * LDSB;   // doubles per B plane
constexpr int SM_STAGE = 2 * SM_PLANE + 2 * SM_PLANEB;   // A_re, A_im, B_re, B_im
constexpr size_t SM_BYTES = 2 * SM_STAGE * sizeof(double);
// Padded request of the chunk pipeline (be_ctx::gemm_pad): 2 x (SM_PAD + 1 KB) exceeds the 228 KB of an
// SM, so at most ONE GEMM CTA is resident per SM, and SM_PAD + one k_hemv CTA (109 KB + 1 KB) still fits:
// the FP64-bound GEMM of one chunk and the HBM-bound k_hemv of the next share every SM.
constexpr size_t SM_PAD = 116 * 1024;

__device__ __forceinline__ void dmma(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

template <int OPA, int OPB, bool PHI, bool SPLIT>
__global__ void __launch_bounds__(NTHREADS, 2) zgemm_kernel(const ZgemmParams p, int tilesM, int tilesN) {
  extern __shared__ double smem[];
  const int tid = threadIdx.x;
  // lower: only the tilesM (tilesM + 1) / 2 tiles on or below the diagonal are launched
  const int64_t tiles = p.lower ? (int64_t)(TM / TN) * tilesM * (tilesM + 1) / 2 : (int64_t)tilesM * tilesN;
  const int64_t bidx = blockIdx.x;
  const int64_t b = bidx / tiles;
  const int t = (int)(bidx - b * tiles);
  int tm, tn;
  if (p.lower) {
    // row tm of TM-row tiles holds RT (tm + 1) tiles of TN columns, RT = TM / TN
    constexpr int RT = TM / TN;
    tm = (int)((sqrt(8.0 * t / RT + 1.0) - 1.0) * 0.5);
    while (RT * (tm + 1) * (tm + 2) / 2 <= t) ++tm;
    while (RT * tm * (tm + 1) / 2 > t) --tm;
    tn = t - RT * tm * (tm + 1) / 2;
  } else { tm = t % tilesM; tn = t / tilesM; }
  const int64_t bo = b / p.inner;
  const int bi = (int)(b - bo * p.inner);
  const cplx* __restrict__ A = p.A + bo * p.sAo + (int64_t)bi * p.sAi;
  int biB = bi;
  bool wrap = false;
  if (p.ringB) { biB = bi + 1; if (biB == p.inner) biB = 0; wrap = (bi == p.phi_at); }
  const cplx* __restrict__ B = p.B + bo * p.sBo + (int64_t)biB * p.sBi;
  cplx* __restrict__ C = p.C + bo * p.sCo + (int64_t)bi * p.sCi;
  const cplx* __restrict__ phi = (PHI && wrap && p.phiB) ? p.phiB : nullptr;
  const int ksplit = SPLIT ? p.ksplit : 0;
  const cplx* __restrict__ A2 = SPLIT ? p.A2 + bo * p.sA2o : nullptr;
  const cplx* __restrict__ B2 = SPLIT ? p.B2 + bo * p.sB2o : nullptr;

  const int m0 = tm * TM, n0 = tn * TN;
  const int M = p.M, N = p.N, K = p.K;
  const bool transA = (OPA == BE_OP_T || OPA == BE_OP_C), conjA = (OPA == BE_OP_C || OPA == BE_OP_J);
  const bool transB = (OPB == BE_OP_T || OPB == BE_OP_C), conjB = (OPB == BE_OP_C || OPB == BE_OP_J);

  // staging coordinates
  int ai, ak, aqi, aqk;   // A tile element (i, k) = (ai + q*aqi, ak + q*aqk), q = 0..QA-1
  if (!transA) { ai = tid % TM; ak = tid / TM; aqi = 0; aqk = NTHREADS / TM; }
  else         { ak = tid % TK; ai = tid / TK; aqi = NTHREADS / TK; aqk = 0; }
  int bn, bk, bqn, bqk;   // B tile element (k, n) = (bk + q*bqk, bn + q*bqn), q = 0..QB-1
  if (!transB) { bk = tid % TK; bn = tid / TK; bqn = NTHREADS / TK; bqk = 0; }
  else         { bn = tid % TN; bk = tid / TN; bqn = 0; bqk = NTHREADS / TN; }

  cplx ra[QA], rb[QB], rphi[QB];
  auto gload = [&](int k0) {
#pragma unroll
    for (int q = 0; q < QA; ++q) {
      const int i = m0 + ai + q * aqi, k = k0 + ak + q * aqk;
      cplx v = mkc(0.0, 0.0);
      if (i < M && k < K) {
        const cplx* Ap = A; int kk = k;
        if (SPLIT && k >= ksplit) { Ap = A2; kk = k - ksplit; }
        v = transA ? Ap[(int64_t)kk + (int64_t)i * p.lda] : Ap[(int64_t)i + (int64_t)kk * p.lda];
      }
      ra[q] = v;
    }
#pragma unroll
    for (int q = 0; q < QB; ++q) {
      const int n = n0 + bn + q * bqn, k = k0 + bk + q * bqk;
      cplx v = mkc(0.0, 0.0);
      cplx f = mkc(1.0, 0.0);
      if (n < N && k < K) {
        const cplx* Bp = B; int kk = k;
        if (SPLIT && k >= ksplit) { Bp = B2; kk = k - ksplit; }
        v = transB ? Bp[(int64_t)n + (int64_t)kk * p.ldb] : Bp[(int64_t)kk + (int64_t)n * p.ldb];
        if (PHI && phi) f = phi[k];
      }
      rb[q] = v;          // no arithmetic on loaded values here: the loads stay in flight during the
      if (PHI) rphi[q] = f;   // multiplication of the current tile; sign flips / phases are applied in sstore
    }
  };
  auto sstore = [&](int stage) {
    double* s = smem + stage * SM_STAGE;
#pragma unroll
    for (int q = 0; q < QA; ++q) {
      const int i = ai + q * aqi, k = ak + q * aqk;
      const int o = transA ? i * LDK + k : k * LDS + i;   // conflict-free for the store and the fragment loads
      s[o] = ra[q].x;
      s[SM_PLANE + o] = conjA ? -ra[q].y : ra[q].y;
    }
#pragma unroll
    for (int q = 0; q < QB; ++q) {
      const int n = bn + q * bqn, k = bk + q * bqk;
      cplx v = rb[q];
      if (PHI) v = cmul(rphi[q], v);
      const int o = transB ? k * LDSB + n : n * LDK + k;
      s[2 * SM_PLANE + o] = v.x;
      s[2 * SM_PLANE + SM_PLANEB + o] = conjB ? -v.y : v.y;
    }
  };

  const int warp = tid >> 5, lane = tid & 31;
  const int wm = warp & 1, wn = warp >> 1;
  const int g = lane >> 2, tg = lane & 3;

  // 4M: accr = Re, acci = Im.  3M: accr = sum Ar Br, acci = sum Ai Bi, accs = sum (Ar + Ai)(Br + Bi).
  double accr[4][2][2], acci[4][2][2], accs[M3 ? 4 : 1][2][2];
#pragma unroll
  for (int a = 0; a < 4; ++a)
#pragma unroll
    for (int c = 0; c < 2; ++c) {
      accr[a][c][0] = accr[a][c][1] = 0.0; acci[a][c][0] = acci[a][c][1] = 0.0;
      if (M3) accs[a][c][0] = accs[a][c][1] = 0.0;
    }

  const bool has_beta = (p.beta.x != 0.0 || p.beta.y != 0.0);
  auto cload = [&](int half, cplx (&dst)[2][2][2]) {
#pragma unroll
    for (int m2 = 0; m2 < 2; ++m2) {
      const int mb = half * 2 + m2;
      const int row = m0 + wm * 32 + mb * 8 + g;
#pragma unroll
      for (int nb = 0; nb < 2; ++nb)
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          const int col = n0 + wn * 16 + nb * 8 + 2 * tg + e;
          dst[m2][nb][e] = (row < M && col < N) ? C[(int64_t)row + (int64_t)col * p.ldc] : mkc(0.0, 0.0);
        }
    }
  };
  const int KT = (K + TK - 1) / TK;
  gload(0);
  sstore(0);
  __syncthreads();
  for (int kt = 0; kt < KT; ++kt) {
    const int cur = kt & 1;
    if (kt + 1 < KT) gload((kt + 1) * TK);
    const double* s = smem + cur * SM_STAGE;
#pragma unroll
    for (int ks = 0; ks < 4; ++ks) {
      const int k = ks * 4 + tg;
      double ar[4], aim[4], br[2], bim[2];
#pragma unroll
      for (int mb = 0; mb < 4; ++mb) {
        const int i = wm * 32 + mb * 8 + g;
        const int o = transA ? i * LDK + k : k * LDS + i;
        ar[mb] = s[o];
        aim[mb] = s[SM_PLANE + o];
      }
#pragma unroll
      for (int nb = 0; nb < 2; ++nb) {
        const int n = wn * 16 + nb * 8 + g;
        const int o = transB ? k * LDSB + n : n * LDK + k;
        br[nb] = s[2 * SM_PLANE + o];
        bim[nb] = s[2 * SM_PLANE + SM_PLANEB + o];
      }
      if (M3) {
        // three real products instead of four (Karatsuba): Re = P1 - P2, Im = P3 - P1 - P2 with P1 = Ar Br,
        // P2 = Ai Bi, P3 = (Ar + Ai)(Br + Bi).  The tensor pipe is the bound of this loop (ncu: math-pipe
        // throttle is the top stall), so a quarter fewer DMMAs is a quarter less main-loop time; the six
        // extra additions per k-step are noise.  Error: normwise eps |A||B| on both parts.
        double sa[4], sb[2];
#pragma unroll
        for (int mb = 0; mb < 4; ++mb) sa[mb] = ar[mb] + aim[mb];
#pragma unroll
        for (int nb = 0; nb < 2; ++nb) sb[nb] = br[nb] + bim[nb];
#pragma unroll
        for (int mb = 0; mb < 4; ++mb)
#pragma unroll
          for (int nb = 0; nb < 2; ++nb) {
            dmma(accr[mb][nb][0], accr[mb][nb][1], ar[mb], br[nb]);
            dmma(acci[mb][nb][0], acci[mb][nb][1], aim[mb], bim[nb]);
            dmma(accs[mb][nb][0], accs[mb][nb][1], sa[mb], sb[nb]);
          }
        continue;
      }
      // four real products; consecutive DMMAs never touch the same accumulator (no back-to-back
      // dependency on the 16-deep accumulator set)
#pragma unroll
      for (int mb = 0; mb < 4; ++mb)
#pragma unroll
        for (int nb = 0; nb < 2; ++nb) {
          dmma(accr[mb][nb][0], accr[mb][nb][1], ar[mb], br[nb]);
          dmma(acci[mb][nb][0], acci[mb][nb][1], ar[mb], bim[nb]);
        }
#pragma unroll
      for (int mb = 0; mb < 4; ++mb) {
        const double nai = -aim[mb];
#pragma unroll
        for (int nb = 0; nb < 2; ++nb) {
          dmma(accr[mb][nb][0], accr[mb][nb][1], nai, bim[nb]);
          dmma(acci[mb][nb][0], acci[mb][nb][1], aim[mb], br[nb]);
        }
      }
    }
    if (kt + 1 < KT) {
      sstore(cur ^ 1);   // the other stage was last read before the previous barrier
      __syncthreads();
    }
  }

  // epilogue in two halves of 8 elements: all loads of C first (independent, in flight together), then the stores -- a load/store per element
  // in program order would serialize 16 round trips
#pragma unroll
  for (int half = 0; half < 2; ++half) {
    cplx cold[2][2][2];
    if (has_beta) {
      cload(half, cold);
    }
#pragma unroll
    for (int m2 = 0; m2 < 2; ++m2) {
      const int mb = half * 2 + m2;
      const int row = m0 + wm * 32 + mb * 8 + g;
#pragma unroll
      for (int nb = 0; nb < 2; ++nb)
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          const int col = n0 + wn * 16 + nb * 8 + 2 * tg + e;
          if (row >= M || col >= N) continue;
          const cplx ab = M3 ? mkc(accr[mb][nb][e] - acci[mb][nb][e], accs[mb][nb][e] - accr[mb][nb][e] - acci[mb][nb][e])
                             : mkc(accr[mb][nb][e], acci[mb][nb][e]);
          cplx v = cmul(p.alpha, ab);
          if (has_beta) v = cadd(v, cmul(p.beta, cold[m2][nb][e]));
          C[(int64_t)row + (int64_t)col * p.ldc] = v;
        }
    }
  }
}


// ---------------------------------------------------------------------------------------------------------
// cp.async variant (no closing phase): the operands stay INTERLEAVED (re, im) in shared memory, one 16-byte
// cp.async per complex element straight from global memory (no staging registers, zero fill at the edges via
// src-size 0), one 16-byte fragment load per operand element.  Transposition is a choice of shared-memory
// layout ([k][mn] with LD % 8 == 2 or [mn][k] with LDK % 8 == 4: both conflict free for the 16-byte fragment
// loads, 8 lanes per wavefront); conjugation is folded into the 3-multiplication algebra
// (Ai -> sA Ai, Bi -> sB Bi: P3 = (Ar + sA Ai)(Br + sB Bi), Re = P1 - sA sB P2, Im = P3 - P1 - sA sB P2 with the
// raw P2 = Ai Bi).  Without the 48 staging registers the kernel fits 168 registers: three CTAs per SM.
constexpr int ALD = TM + 2, BLD = TN + 2;
constexpr int AS_A = (TM * LDK > TK * ALD) ? TM * LDK : TK * ALD;
constexpr int AS_B = (TN * LDK > TK * BLD) ? TN * LDK : TK * BLD;
constexpr int AS_STAGE = AS_A + AS_B;                       // complex elements per stage
constexpr size_t AS_BYTES = 2 * AS_STAGE * sizeof(cplx);

__device__ __forceinline__ void cp_async16(const cplx* smem_dst, const cplx* gsrc, bool pred) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  const int sz = pred ? 16 : 0;
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" :: "r"(d), "l"(gsrc), "r"(sz) : "memory");
}

template <int OPA, int OPB, bool SPLIT>
__global__ void __launch_bounds__(NTHREADS, 3) zgemm_async_kernel(const ZgemmParams p, int tilesM, int tilesN) {
  extern __shared__ __align__(16) double smem[];
  cplx* sm = reinterpret_cast<cplx*>(smem);
  const int tid = threadIdx.x;
  const int64_t tiles = p.lower ? (int64_t)(TM / TN) * tilesM * (tilesM + 1) / 2 : (int64_t)tilesM * tilesN;
  const int64_t bidx = blockIdx.x;
  const int64_t b = bidx / tiles;
  const int t = (int)(bidx - b * tiles);
  int tm, tn;
  if (p.lower) {
    constexpr int RT = TM / TN;
    tm = (int)((sqrt(8.0 * t / RT + 1.0) - 1.0) * 0.5);
    while (RT * (tm + 1) * (tm + 2) / 2 <= t) ++tm;
    while (RT * tm * (tm + 1) / 2 > t) --tm;
    tn = t - RT * tm * (tm + 1) / 2;
  } else { tm = t % tilesM; tn = t / tilesM; }
  const int64_t bo = b / p.inner;
  const int bi = (int)(b - bo * p.inner);
  const cplx* __restrict__ A = p.A + bo * p.sAo + (int64_t)bi * p.sAi;
  int biB = bi;
  if (p.ringB) { biB = bi + 1; if (biB == p.inner) biB = 0; }
  const cplx* __restrict__ B = p.B + bo * p.sBo + (int64_t)biB * p.sBi;
  cplx* __restrict__ C = p.C + bo * p.sCo + (int64_t)bi * p.sCi;
  const int ksplit = SPLIT ? p.ksplit : 0;
  const cplx* __restrict__ A2 = SPLIT ? p.A2 + bo * p.sA2o : nullptr;
  const cplx* __restrict__ B2 = SPLIT ? p.B2 + bo * p.sB2o : nullptr;

  const int m0 = tm * TM, n0 = tn * TN;
  const int M = p.M, N = p.N, K = p.K;
  constexpr bool transA = (OPA == BE_OP_T || OPA == BE_OP_C), conjA = (OPA == BE_OP_C || OPA == BE_OP_J);
  constexpr bool transB = (OPB == BE_OP_T || OPB == BE_OP_C), conjB = (OPB == BE_OP_C || OPB == BE_OP_J);

  int ai, ak, aqi, aqk;
  if (!transA) { ai = tid % TM; ak = tid / TM; aqi = 0; aqk = NTHREADS / TM; }
  else         { ak = tid % TK; ai = tid / TK; aqi = NTHREADS / TK; aqk = 0; }
  int bn, bk, bqn, bqk;
  if (!transB) { bk = tid % TK; bn = tid / TK; bqn = NTHREADS / TK; bqk = 0; }
  else         { bn = tid % TN; bk = tid / TN; bqn = 0; bqk = NTHREADS / TN; }

  auto aload = [&](int k0, int stage) {
    cplx* sa_ = sm + stage * AS_STAGE;
    cplx* sb_ = sa_ + AS_A;
#pragma unroll
    for (int q = 0; q < QA; ++q) {
      const int il = ai + q * aqi, kl = ak + q * aqk;
      const int i = m0 + il, k = k0 + kl;
      const bool ok = (i < M && k < K);
      const cplx* Ap = A; int kk = k;
      if (SPLIT && k >= ksplit) { Ap = A2; kk = k - ksplit; }
      const cplx* src = ok ? (transA ? Ap + (int64_t)kk + (int64_t)i * p.lda : Ap + (int64_t)i + (int64_t)kk * p.lda) : A;
      cp_async16(sa_ + (transA ? il * LDK + kl : kl * ALD + il), src, ok);
    }
#pragma unroll
    for (int q = 0; q < QB; ++q) {
      const int nl = bn + q * bqn, kl = bk + q * bqk;
      const int n = n0 + nl, k = k0 + kl;
      const bool ok = (n < N && k < K);
      const cplx* Bp = B; int kk = k;
      if (SPLIT && k >= ksplit) { Bp = B2; kk = k - ksplit; }
      const cplx* src = ok ? (transB ? Bp + (int64_t)n + (int64_t)kk * p.ldb : Bp + (int64_t)kk + (int64_t)n * p.ldb) : B;
      cp_async16(sb_ + (transB ? kl * BLD + nl : nl * LDK + kl), src, ok);
    }
    asm volatile("cp.async.commit_group;\n" ::: "memory");
  };

  const int warp = tid >> 5, lane = tid & 31;
  const int wm = warp & 1, wn = warp >> 1;
  const int g = lane >> 2, tg = lane & 3;

  double accr[4][2][2], acci[4][2][2], accs[4][2][2];
#pragma unroll
  for (int a = 0; a < 4; ++a)
#pragma unroll
    for (int c = 0; c < 2; ++c) {
      accr[a][c][0] = accr[a][c][1] = 0.0; acci[a][c][0] = acci[a][c][1] = 0.0; accs[a][c][0] = accs[a][c][1] = 0.0;
    }

  const int KT = (K + TK - 1) / TK;
  const bool has_beta = (p.beta.x != 0.0 || p.beta.y != 0.0);
  aload(0, 0);
  if (has_beta) {
    // read-modify-write (the rank-2k update has only K / TK = 4 k-tiles per C tile): pull the C tile, 32 columns
    // of 1 KB, into L2 now so that the epilogue's loads do not wait on DRAM
#pragma unroll
    for (int q = 0; q < TM * TN * 16 / 128 / NTHREADS; ++q) {
      const int line = tid + q * NTHREADS;
      const int col = n0 + line / (TM / 8), row = m0 + (line % (TM / 8)) * 8;
      if (row < M && col < N) asm volatile("prefetch.global.L2 [%0];\n" :: "l"(C + (int64_t)row + (int64_t)col * p.ldc));
    }
  }
  for (int kt = 0; kt < KT; ++kt) {
    const int cur = kt & 1;
    asm volatile("cp.async.wait_group 0;\n" ::: "memory");
    __syncthreads();                 // tile kt visible to all; everyone is done with tile kt-1 (the other stage)
    if (kt + 1 < KT) aload((kt + 1) * TK, cur ^ 1);
    const cplx* sA_ = sm + cur * AS_STAGE;
    const cplx* sB_ = sA_ + AS_A;
#pragma unroll
    for (int ks = 0; ks < 4; ++ks) {
      const int k = ks * 4 + tg;
      cplx a[4], bb[2];
#pragma unroll
      for (int mb = 0; mb < 4; ++mb) {
        const int i = wm * 32 + mb * 8 + g;
        a[mb] = sA_[transA ? i * LDK + k : k * ALD + i];
      }
#pragma unroll
      for (int nb = 0; nb < 2; ++nb) {
        const int n = wn * 16 + nb * 8 + g;
        bb[nb] = sB_[transB ? k * BLD + n : n * LDK + k];
      }
      double sa[4], sb[2];
#pragma unroll
      for (int mb = 0; mb < 4; ++mb) sa[mb] = conjA ? a[mb].x - a[mb].y : a[mb].x + a[mb].y;
#pragma unroll
      for (int nb = 0; nb < 2; ++nb) sb[nb] = conjB ? bb[nb].x - bb[nb].y : bb[nb].x + bb[nb].y;
#pragma unroll
      for (int mb = 0; mb < 4; ++mb)
#pragma unroll
        for (int nb = 0; nb < 2; ++nb) {
          dmma(accr[mb][nb][0], accr[mb][nb][1], a[mb].x, bb[nb].x);
          dmma(acci[mb][nb][0], acci[mb][nb][1], a[mb].y, bb[nb].y);
          dmma(accs[mb][nb][0], accs[mb][nb][1], sa[mb], sb[nb]);
        }
    }
  }

  constexpr double ss = (conjA != conjB) ? -1.0 : 1.0;   // sA sB
#pragma unroll
  for (int half = 0; half < 2; ++half) {
    cplx cold[2][2][2];
    if (has_beta) {
#pragma unroll
      for (int m2 = 0; m2 < 2; ++m2) {
        const int row = m0 + wm * 32 + (half * 2 + m2) * 8 + g;
#pragma unroll
        for (int nb = 0; nb < 2; ++nb)
#pragma unroll
          for (int e = 0; e < 2; ++e) {
            const int col = n0 + wn * 16 + nb * 8 + 2 * tg + e;
            cold[m2][nb][e] = (row < M && col < N) ? C[(int64_t)row + (int64_t)col * p.ldc] : mkc(0.0, 0.0);
          }
      }
    }
#pragma unroll
    for (int m2 = 0; m2 < 2; ++m2) {
      const int mb = half * 2 + m2;
      const int row = m0 + wm * 32 + mb * 8 + g;
#pragma unroll
      for (int nb = 0; nb < 2; ++nb)
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          const int col = n0 + wn * 16 + nb * 8 + 2 * tg + e;
          if (row >= M || col >= N) continue;
          const double p2 = ss * acci[mb][nb][e];
          const cplx ab = mkc(accr[mb][nb][e] - p2, accs[mb][nb][e] - accr[mb][nb][e] - p2);
          cplx v = cmul(p.alpha, ab);
          if (has_beta) v = cadd(v, cmul(p.beta, cold[m2][nb][e]));
          C[(int64_t)row + (int64_t)col * p.ldc] = v;
        }
    }
  }
}

static int gemm_async_mode() {   // BE_GEMM_ASYNC=0 selects the register-staged kernel everywhere (A/B measurements)
  const char* e = getenv("BE_GEMM_ASYNC");
  return (e && e[0] == '0') ? 0 : 1;
}

template <int OPA, int OPB, bool PHI, bool SPLIT>
int launch(be_ctx* ctx, const ZgemmParams& p) {
  const int tilesM = (p.M + TM - 1) / TM, tilesN = (p.N + TN - 1) / TN;
  if (p.lower && p.M != p.N) return BE_ERR_SHAPE;
  const int64_t blocks = p.batch * (p.lower ? (int64_t)(TM / TN) * tilesM * (tilesM + 1) / 2 : (int64_t)tilesM * tilesN);
  if (blocks <= 0) return BE_OK;
  if (blocks > 0x7fffffffLL) return BE_ERR_SHAPE;
  // function attributes are per device: set on every launch (the context's device is current; no process-wide flag)
  be_prof_begin(ctx, PK_GEMM);
  if constexpr (!PHI) {
    if (M3 && gemm_async_mode() && !ctx->gemm_pad) {
      BE_CUDA(cudaFuncSetAttribute(zgemm_async_kernel<OPA, OPB, SPLIT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)AS_BYTES));
      BE_CUDA(cudaFuncSetAttribute(zgemm_async_kernel<OPA, OPB, SPLIT>, cudaFuncAttributePreferredSharedMemoryCarveout, 100));
      zgemm_async_kernel<OPA, OPB, SPLIT><<<(unsigned)blocks, NTHREADS, AS_BYTES, ctx->stream>>>(p, tilesM, tilesN);
    } else {
      BE_CUDA(cudaFuncSetAttribute(zgemm_kernel<OPA, OPB, PHI, SPLIT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SM_PAD));
      zgemm_kernel<OPA, OPB, PHI, SPLIT><<<(unsigned)blocks, NTHREADS, (ctx->gemm_pad && ctx->stream == ctx->stream2) ? SM_PAD : SM_BYTES, ctx->stream>>>(p, tilesM, tilesN);
    }
  } else {
    BE_CUDA(cudaFuncSetAttribute(zgemm_kernel<OPA, OPB, PHI, SPLIT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SM_PAD));
    zgemm_kernel<OPA, OPB, PHI, SPLIT><<<(unsigned)blocks, NTHREADS, (ctx->gemm_pad && ctx->stream == ctx->stream2) ? SM_PAD : SM_BYTES, ctx->stream>>>(p, tilesM, tilesN);
  }
  {
    const double tri = p.lower ? 0.5 : 1.0;
    const double fl = 8.0 * p.M * (double)p.N * p.K * (double)p.batch * tri;
    const double by = 16.0 * (double)p.batch * ((double)p.M * p.K + (double)p.K * p.N + tri * (double)p.M * p.N * (1.0 + (p.beta.x != 0.0 || p.beta.y != 0.0)));
    be_prof_end(ctx, PK_GEMM, by, fl);
  }
  ctx->launches++;
  return (int)cudaGetLastError();
}

}  // namespace

int be_zgemm(be_ctx* ctx, int opA, int opB, const ZgemmParams& p) {
  if (p.M <= 0 || p.N <= 0 || p.batch <= 0) return BE_OK;
  if (p.phiB && (opA != BE_OP_C || opB != BE_OP_N || !p.ringB)) return BE_ERR_UNSUPPORTED;   // closing phase: link GEMM only
  if (p.phiB && p.ringB) return launch<BE_OP_C, BE_OP_N, true, false>(ctx, p);
  if (p.ksplit > 0) {   // two K segments: the rank-2k update only
    if (opA != BE_OP_N || opB != BE_OP_C || !p.A2 || !p.B2) return BE_ERR_UNSUPPORTED;
    return launch<BE_OP_N, BE_OP_C, false, true>(ctx, p);
  }
#define CASE(a, b) if (opA == a && opB == b) return launch<a, b, false, false>(ctx, p);
  CASE(BE_OP_N, BE_OP_N) CASE(BE_OP_N, BE_OP_C) CASE(BE_OP_C, BE_OP_N) CASE(BE_OP_N, BE_OP_T)
  CASE(BE_OP_T, BE_OP_N) CASE(BE_OP_J, BE_OP_N) CASE(BE_OP_N, BE_OP_J) CASE(BE_OP_C, BE_OP_C) CASE(BE_OP_T, BE_OP_J)
#undef CASE
  return BE_ERR_UNSUPPORTED;
}
