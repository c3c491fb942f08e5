// be_wilson_loop / be_spin_resolved_wilson / be_nested_wilson and their host-buffer variants:
// chunking over whole loops and stage sequencing.
#include "be_common.cuh"
#include <string.h>
#include <math.h>
#include <vector>
#include <algorithm>

int be_mingap(be_ctx* ctx, const double* E, int N, int lo, int hi, int n1, int64_t loops, double* out);
int be_scale_rows(be_ctx* ctx, const cplx* X, const double* S, cplx* SX, int N, int64_t total);
int be_pack_rows(be_ctx* ctx, const cplx* X, const double* S, const int* sel, double b, cplx* XA, cplx* SXA, int N,
                 int nsel, int64_t cols);
int be_add_diag(be_ctx* ctx, cplx* A, int m, int64_t cnt, double b);
int be_flag_loops(be_ctx* ctx, const int* info, const double* E, int ldE, int n1, int64_t nl, int* bad0, int* bad1);
int be_nested_select_small(be_ctx* ctx, const cplx* W, int64_t cnt, int m, int wb_lo, int wb_hi,
                           double cut, double* theta1, cplx* Vs);
int be_chain_product(be_ctx* ctx, const cplx* F, int N, int m, int64_t outer, int n1,
                     const cplx* d_close, int phi_at, cplx* Wdst, cplx** Wout);

static inline bool aligned(const void* p, size_t a) { return ((uintptr_t)p % a) == 0; }

static int make_map(const be_grid* g, int dir, GridMap* out) {
  if (!g) return BE_ERR_NULL;
  if (g->ndim < 1 || g->ndim > 3 || g->batch < 1 || g->N < 1) return BE_ERR_SHAPE;
  if (dir < 0 || dir >= g->ndim) return BE_ERR_SHAPE;
  GridMap m;
  memset(&m, 0, sizeof(m));
  m.ndim = g->ndim; m.dir = dir; m.shift = 0;
  int64_t st = 1, loops = g->batch;
  for (int a = g->ndim - 1; a >= 0; --a) {
    if (g->dims[a] < 1) return BE_ERR_SHAPE;
    m.dims[a] = g->dims[a]; m.stride[a] = st; st *= g->dims[a];
    if (a != dir) loops *= g->dims[a];
  }
  m.batch_stride = st; m.n1 = g->dims[dir]; m.loops = loops;
  *out = m;
  return BE_OK;
}

// host grids: matrices of at least this order are copied as row blocks of their upper triangle
constexpr int HOST_TRI_MINN = 256, HOST_TRI_BLOCKS = 8;

struct SpinArgs {
  const void* dS; int S_is_diag; int m_lo;
  double* theta_lo; double* theta_hi; double* pso;
  // diagonal S whose most frequent value bval sits on at least half of the rows (set by analyze_diag_S):
  // sel [nsel] = the other rows, ascending (device)
  const int* sel; int nsel; double bval;
};

// bytes of scratch one loop needs (upper bound), plain or spin-resolved
static size_t per_loop_bytes(int N, int m, int n1, bool spin, int lo = 0) {
  const size_t fr = (size_t)N * m * sizeof(cplx);
  // a band window [lo, lo + m) needs the lowest lo + m vectors, then a compact copy of its m columns
  size_t b = (size_t)n1 * (be_eigh_scratch_bytes(1, N, lo + m) + (size_t)N * (lo + m) * sizeof(cplx) + (lo ? fr : 0) +
                           (size_t)N * sizeof(double) + 512);
  const size_t mm = (size_t)m * m * sizeof(cplx);
  b += (size_t)2 * n1 * mm + 8 * mm + (size_t)m * 64 + 4096;       // links, product tree, eigenvalues
  if (spin) {
    b += (size_t)n1 * (fr /*SX*/ + 2 * mm /*S_red, V*/ + fr /*sector frames*/ + (size_t)m * 8 + 1024);
    const size_t inner = (size_t)n1 * be_eigh_scratch_bytes(1, m, m);
    const size_t outer = (size_t)n1 * be_eigh_scratch_bytes(1, N, m);
    if (inner > outer) b += inner - outer;
  }
  return b;
}

// S6, first half: S_red = U^H S U for cnt frames X, S_red = V Sigma V^H (ascending).
// pso_out [cnt][m] receives Sigma (or scratch when NULL); *Vout [cnt][m][m] column-major.
static int pso_eigenvectors(be_ctx* ctx, const cplx* X, int64_t cnt, int N, int m, const SpinArgs* sp,
                            double* pso_out, cplx** Vout, int* info, double** sig_out) {
  const bool packed = sp->S_is_diag && sp->sel != nullptr;
  const int ks = packed ? sp->nsel : N;    // rows that enter the contraction
  cplx* SX = (cplx*)be_arena_alloc(ctx, (size_t)cnt * ks * m * sizeof(cplx));
  cplx* XA = packed ? (cplx*)be_arena_alloc(ctx, (size_t)cnt * ks * m * sizeof(cplx)) : nullptr;
  cplx* Sred = (cplx*)be_arena_alloc(ctx, (size_t)cnt * m * m * sizeof(cplx));
  cplx* V = (cplx*)be_arena_alloc(ctx, (size_t)cnt * m * m * sizeof(cplx));
  double* sig = pso_out ? pso_out : (double*)be_arena_alloc(ctx, (size_t)cnt * m * sizeof(double));
  if (!SX || !Sred || !V || !sig || (packed && !XA)) return BE_ERR_NOMEM;
  if (packed) {
    // U^H S U = b I + U_A^H (S_A - b) U_A (U^H U = I): only the rows with S != b enter the GEMM
    BE_TRY(be_pack_rows(ctx, X, (const double*)sp->dS, sp->sel, sp->bval, XA, SX, N, ks, cnt * (int64_t)m));
  } else if (sp->S_is_diag) {
    BE_TRY(be_scale_rows(ctx, X, (const double*)sp->dS, SX, N, cnt * (int64_t)N * m));
  } else {
    // row-major S read column-major is S^T: op T recovers S;  SX = S X
    ZgemmParams g = zgemm_simple(N, m, N, (const cplx*)sp->dS, N, 0, X, N, (int64_t)N * m,
                                 SX, N, (int64_t)N * m, cnt);
    BE_TRY(be_zgemm(ctx, BE_OP_T, BE_OP_N, g));
  }
  if (ks > 0) {
    // the eigensolver reads its input row-major; a column-major buffer holding conj(S_red) =
    // X^T conj(SX) is S_red when read row-major (S_red is Hermitian)
    ZgemmParams g = zgemm_simple(m, m, ks, packed ? XA : X, ks, (int64_t)ks * m, SX, ks, (int64_t)ks * m,
                                 Sred, m, (int64_t)m * m, cnt);
    g.lower = 1;   // the eigensolver reads only the lower triangle of the column-major buffer
    BE_TRY(be_zgemm(ctx, BE_OP_T, BE_OP_J, g));
  } else {
    BE_CUDA(cudaMemsetAsync(Sred, 0, (size_t)cnt * m * m * sizeof(cplx), ctx->stream));
  }
  if (packed) BE_TRY(be_add_diag(ctx, Sred, m, cnt, sp->bval));
  GridMap fm;
  memset(&fm, 0, sizeof(fm));
  fm.ndim = 1; fm.dir = 0; fm.n1 = 1; fm.dims[0] = 1; fm.batch_stride = 1; fm.loops = cnt;
  BE_TRY(be_eigh_frames(ctx, Sred, fm, 0, cnt, m, m, m, sig, V, info));
  *Vout = V;
  if (sig_out) *sig_out = sig;
  return BE_OK;
}

static int wilson_chunk(be_ctx* ctx, const cplx* H, const GridMap& map, int64_t gl0, int N, int m, int n1, int64_t l0,
                        int64_t nl, int64_t cnt, const cplx* d_close, double* d_mingap, const SpinArgs* sp, int mlo,
                        int mhi, cplx* const* Wall, int* bad, int64_t loops);

static int pipeline_init(be_ctx* ctx) {
  if (ctx->stream2) return BE_OK;
  int least = 0, greatest = 0;
  BE_CUDA(cudaDeviceGetStreamPriorityRange(&least, &greatest));
  BE_CUDA(cudaStreamCreateWithPriority(&ctx->stream2, cudaStreamNonBlocking, greatest));
  BE_CUDA(cudaEventCreateWithFlags(&ctx->ev_split, cudaEventDisableTiming));
  BE_CUDA(cudaEventCreateWithFlags(&ctx->ev_join, cudaEventDisableTiming));
  BE_CUDA(cudaEventCreateWithFlags(&ctx->ev_region[0], cudaEventDisableTiming));
  BE_CUDA(cudaEventCreateWithFlags(&ctx->ev_region[1], cudaEventDisableTiming));
  return BE_OK;
}

// Diagonal S: find its most frequent value b; when at least half of the rows carry it, pso_eigenvectors
// contracts only over the other rows (list written to d_sel).  One small device -> host copy per call.
static int analyze_diag_S(be_ctx* ctx, SpinArgs* sp, int N, int* d_sel) {
  std::vector<double> h((size_t)N);
  BE_CUDA(cudaMemcpyAsync(h.data(), sp->dS, (size_t)N * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
  BE_CUDA(cudaStreamSynchronize(ctx->stream));
  for (int r = 0; r < N; ++r) if (!(h[r] == h[r])) return BE_OK;   // NaN: leave it to the general path
  std::vector<double> srt(h);
  std::sort(srt.begin(), srt.end());
  double b = srt[0];
  int best = 0;
  for (int i = 0; i < N;) {
    int j = i;
    while (j < N && srt[j] == srt[i]) ++j;
    if (j - i > best) { best = j - i; b = srt[i]; }
    i = j;
  }
  if (2 * best < N) return BE_OK;
  std::vector<int> sel;
  for (int r = 0; r < N; ++r) if (h[r] != b) sel.push_back(r);
  if (!sel.empty()) {
    BE_CUDA(cudaMemcpyAsync(d_sel, sel.data(), sel.size() * sizeof(int), cudaMemcpyHostToDevice, ctx->stream));
    BE_CUDA(cudaStreamSynchronize(ctx->stream));   // sel is a local
  }
  sp->sel = d_sel; sp->nsel = (int)sel.size(); sp->bval = b;
  return BE_OK;
}

// One pass over all loops of ``map`` (device H).  Plain loop when ``sp`` is NULL.
static int wilson_device(be_ctx* ctx, const cplx* H, const GridMap& map, int N, int m,
                         const cplx* d_close, double* d_theta, double* d_abs, double* d_mingap,
                         const SpinArgs* sp, HostStage* hs = nullptr, const BlochSrc* bs = nullptr) {
  const int n1 = map.n1;
  const int64_t loops = map.loops;
  // tiny matrices, at most two bands: the whole path in one kernel, a warp per loop (small_loop.cu)
  if (!hs && !bs && ctx->band_lo == 0 && be_small_loop_applies(N, m, n1) && (!sp || sp->m_lo <= m)) {
    if (sp) return be_small_loop(ctx, H, nullptr, map, N, m, d_close, n1 - 1, nullptr, nullptr, nullptr, nullptr, nullptr, sp->dS,
                                 sp->S_is_diag, sp->m_lo, sp->theta_lo, sp->theta_hi, sp->pso);
    return be_small_loop(ctx, H, nullptr, map, N, m, d_close, n1 - 1, d_theta, d_abs, d_mingap, nullptr, nullptr, nullptr, 0, 0,
                         nullptr, nullptr, nullptr);
  }
  be_subspace_guard subspace(ctx);   // frames enter only through their span
  SpinArgs spl;
  if (sp) { spl = *sp; spl.sel = nullptr; spl.nsel = 0; spl.bval = 0.0; sp = &spl; }
  const size_t per = per_loop_bytes(N, m, n1, sp != nullptr, ctx->band_lo);
  size_t ws = be_effective_ws_limit(ctx, per * (size_t)loops + (hs ? 2 * hs->loop_bytes * (size_t)loops : 0), hs != nullptr);
  size_t ws_total = ws;   // host grid: scratch arena + the two staging buffers
  if (hs) {
    // the two staging buffers of a host grid come out of the same budget (2 x loop_bytes per loop of a chunk)
    ws_total = ws + ctx->stage_cap[0] + ctx->stage_cap[1];
    ws = (size_t)((double)ws_total * (double)per / (double)(per + 2 * hs->loop_bytes));
  }
  int64_t lc = (int64_t)(ws / per);
  if (lc < 1) lc = 1;
  if (lc > loops) lc = loops;
  // Chunk boundaries.  Device grid: equal chunks of at most lc loops.  Host grid: the first copy cannot overlap
  // anything, so the chunks grow -- 1/8 of the loops, then 1/4, then what the cap allows -- and every later
  // copy hides behind the (longer) computation of the chunk before it.
  std::vector<int64_t> cstart;
  std::vector<int64_t> feed_sub;   // host grid streamed into one chunk: loop boundaries of the sub-ranges
  if (!hs) {
    const int64_t nch = (loops + lc - 1) / lc;
    lc = (loops + nch - 1) / nch;
    for (int64_t l0 = 0; l0 < loops; l0 += lc) cstart.push_back(l0);
  } else {
    // Sizes: the one-CTA-per-matrix kernels of the eigensolver (panel QR, bulge chasing) run in waves of sm_count
    // matrices, so chunks of just under 1, 2, 3, .. waves (5, 8, 11 loops of 25 points on 148 SMs), ascending;
    // matrices too small for that to matter: 1/8 of the loops, then doubling.
    std::vector<int64_t> sz;
    const int64_t w1 = ctx->sm_count / n1;
    if (N > TS_MAXN && w1 >= 1 && w1 < loops) {
      int64_t left = loops;
      for (int k = 1; left > 0; ++k) {
        int64_t c = (int64_t)k * ctx->sm_count / n1;
        if (c > lc) c = lc;
        if (c > left) c = left;
        sz.push_back(c);
        left -= c;
      }
      std::sort(sz.begin(), sz.end());
    } else {
      int64_t left = loops, step = (loops + 7) / 8;
      while (left > 0) {
        int64_t c = step < lc ? step : lc;
        if (left - c > 0 && left - c < c / 2) c = left;   // no tiny last chunk
        if (c > lc) c = lc;
        if (c > left) c = left;
        sz.push_back(c);
        left -= c;
        step *= 2;
      }
    }
    // Large matrices: a loop takes r ~ 5.3 N / 1600 times longer to process than to copy (measured at N = 1600 on
    // PCIe 5: 99 ms against 18.6 ms), and every extra chunk costs the latency-bound stages another round: TWO
    // chunks, the first just long enough to hide the copy of the second, c1 = loops / (1 + r) (24 loops of
    // N = 1600: 4 + 20, 2546 ms against 2604 ms for 5 + 8 + 11 and 2822 ms for one chunk).
    if (N >= 800 && sz.size() >= 2) {
      // (only the upper triangle travels: (HOST_TRI_BLOCKS + 1) / (2 HOST_TRI_BLOCKS) of the bytes)
      const double r = 5.3 * (double)N / 1600.0 * (2.0 * HOST_TRI_BLOCKS) / (HOST_TRI_BLOCKS + 1.0);
      int64_t c1 = (int64_t)ceil((double)loops / (1.0 + r));
      if (c1 < 1) c1 = 1;
      // memory: scratch for the larger chunk, one staging buffer per chunk
      const size_t need2 = per * (size_t)(loops - c1) + (size_t)loops * hs->loop_bytes + ((size_t)1 << 30);   // + persistent part
      if (c1 < loops && need2 <= ws_total) { sz.clear(); sz.push_back(c1); sz.push_back(loops - c1); }
    }
    // Two-stage eigensolver and room for every loop at once: ONE chunk, fed in three sub-ranges (HostFeed).  Only
    // stage 1 of the eigensolver (dense -> band, a third of the pass, throughput bound) runs per sub-range, while
    // the next one travels; everything else sees the whole batch, so nothing pays for small batches.  Stage 1 of a
    // loop takes rho ~ 2.3 N / 1600 times as long as its copy: sub-ranges in the ratio 1 : rho : rho^2
    // (24 loops of N = 1600: 3 + 7 + 14; exposed: the first 3 loops, 31 ms).
    const bool two_stage = N >= BE_BAND_MINN && N <= BE_BAND_MAXN && N > TS_MAXN && !bs &&
                           (ctx->eigh_algo == 1 || (ctx->eigh_algo == 2 && N >= BE_BAND_AUTON));
    if (two_stage && loops >= 3 && sz.size() >= 2) {
      double rho = 2.3 * (double)N / 1600.0;
      rho = rho < 1.2 ? 1.2 : (rho > 3.0 ? 3.0 : rho);
      int64_t s0 = (int64_t)floor((double)loops / (1.0 + rho + rho * rho) + 0.5);
      if (s0 < 1) s0 = 1;
      int64_t s1 = (int64_t)floor((double)s0 * rho + 0.5);
      if (s1 < 1) s1 = 1;
      if (s0 + s1 >= loops) { s0 = 1; s1 = 1; }
      const int64_t s2 = loops - s0 - s1;
      const size_t stg = (size_t)((s0 > s2 ? s0 : s2) + s1) * hs->loop_bytes;
      if (per * (size_t)loops + stg + ((size_t)1 << 30) <= ws_total) {
        feed_sub.push_back(0); feed_sub.push_back(s0); feed_sub.push_back(s0 + s1); feed_sub.push_back(loops);
        sz.clear(); sz.push_back(loops);
      }
    }
    int64_t l0 = 0;
    for (size_t i = 0; i < sz.size(); ++i) { cstart.push_back(l0); l0 += sz[i]; }
    lc = 0;
    for (size_t i = 0; i < cstart.size(); ++i) {
      const int64_t e = (i + 1 < cstart.size()) ? cstart[i + 1] : loops;
      if (e - cstart[i] > lc) lc = e - cstart[i];
    }
  }
  cstart.push_back(loops);
  const int64_t nchunks = (int64_t)cstart.size() - 1;
  const int mlo = sp ? sp->m_lo : 0, mhi = sp ? m - sp->m_lo : 0;
  // The Wilson matrices of ALL loops outlive the chunks: their eigenphase solve (S4) is a
  // latency-bound kernel with one CTA per matrix, so it runs once over every loop at the end
  // instead of once per chunk with a fraction of the SMs busy.
  const int msec[2] = {sp ? mlo : m, sp ? mhi : 0};
  size_t persist = 0;
  for (int s = 0; s < 2; ++s)
    persist += be_align256((size_t)loops * msec[s] * msec[s] * sizeof(cplx)) + be_eigenphases_scratch_bytes(2 * loops, msec[s]) +
               be_align256(2 * (size_t)loops * msec[s] * sizeof(double)) + be_align256(2 * (size_t)loops * sizeof(int)) + 1024;
  persist += be_align256((size_t)N * sizeof(int));
  // Chunk pipeline (more than one chunk): two scratch regions used alternately, the
  // tridiagonalization of chunk c+1 on the caller's stream overlaps the rest of chunk c on stream2.
  const size_t region = be_align256(per * (size_t)lc);
  bool pipe = nchunks > 1 && ctx->chunk_pipeline && !hs;
  // host-resident grid: two staging buffers (kept in the context between calls) next to the work arena
  GridMap smap;
  auto issue_copy = [&](int64_t ci) -> int {
    const int b = (int)(ci & 1);
    const std::vector<int64_t>& cb = feed_sub.empty() ? cstart : feed_sub;   // chunks, or the sub-ranges of the one chunk
    const int64_t c0 = cb[ci], cn = cb[ci + 1] - c0;
    if (ci >= 2) BE_CUDA(cudaStreamWaitEvent(ctx->copy_stream, hs->freed[b], 0));
    const GridMap& hm = hs->hmap;
    if (N >= HOST_TRI_MINN) {
      // The eigensolver reads only the row-major UPPER triangle of a Hermitian H (tests: the other triangle may
      // hold anything): each matrix travels as HOST_TRI_BLOCKS row blocks, block b with the columns from its first
      // row on -- 56 % of the bytes for 8 blocks.  The rest of the staging buffer keeps stale data.
      // One 3D copy per row block covers that block of EVERY matrix of a run of equally spaced matrices (a slice =
      // a matrix): 8 copies per chunk when the loops are contiguous in the host grid, else 8 per loop.  (One 2D
      // copy per matrix and block -- 4000 calls for 500 matrices -- overflows the stream's queue and blocks the
      // host thread until most of the copy is done, before it gets to launch the kernels of the chunk in front.)
      const size_t pitch = (size_t)N * sizeof(cplx);
      const int h = (N + HOST_TRI_BLOCKS - 1) / HOST_TRI_BLOCKS;
      const bool contig = hm.dir == hm.ndim - 1;
      const int64_t runs = contig ? 1 : cn;
      for (int64_t l = 0; l < runs; ++l) {
        const int64_t src = gridmap_index(hm, c0 + l, 0);
        const size_t depth = contig ? (size_t)(cn * n1) : (size_t)n1;
        const size_t src_rows = contig ? (size_t)N : (size_t)hm.stride[hm.dir] * N;   // rows from one matrix to the next
        for (int r0 = 0; r0 < N; r0 += h) {
          const int rows = (N - r0 < h) ? N - r0 : h;
          cudaMemcpy3DParms q;
          memset(&q, 0, sizeof(q));
          q.srcPtr = make_cudaPitchedPtr((void*)(hs->hH + (size_t)src * hs->mat_bytes), pitch, pitch, src_rows);
          q.dstPtr = make_cudaPitchedPtr((char*)hs->stage[b] + (size_t)l * hs->loop_bytes, pitch, pitch, (size_t)N);
          q.srcPos = make_cudaPos((size_t)r0 * sizeof(cplx), (size_t)r0, 0);
          q.dstPos = q.srcPos;
          q.extent = make_cudaExtent((size_t)(N - r0) * sizeof(cplx), (size_t)rows, depth);
          q.kind = cudaMemcpyHostToDevice;
          BE_CUDA(cudaMemcpy3DAsync(&q, ctx->copy_stream));
          ctx->h2d_bytes += (int64_t)(N - r0) * (int64_t)sizeof(cplx) * rows * (int64_t)depth;
        }
      }
    } else if (hm.dir == hm.ndim - 1) {
      // loops are contiguous in the host grid, and so are consecutive loops: one copy per chunk
      BE_CUDA(cudaMemcpyAsync(hs->stage[b], hs->hH + (size_t)c0 * hs->loop_bytes, (size_t)cn * hs->loop_bytes,
                              cudaMemcpyHostToDevice, ctx->copy_stream));
      ctx->h2d_bytes += (int64_t)cn * (int64_t)hs->loop_bytes;
    } else {
      // a loop is n1 matrices a fixed stride apart: one strided copy per loop
      for (int64_t l = 0; l < cn; ++l) {
        const int64_t src = gridmap_index(hm, c0 + l, 0);
        BE_CUDA(cudaMemcpy2DAsync((char*)hs->stage[b] + (size_t)l * hs->loop_bytes, hs->mat_bytes,
                                  hs->hH + (size_t)src * hs->mat_bytes, (size_t)hm.stride[hm.dir] * hs->mat_bytes,
                                  hs->mat_bytes, (size_t)n1, cudaMemcpyHostToDevice, ctx->copy_stream));
        ctx->h2d_bytes += (int64_t)hs->loop_bytes;
      }
    }
    BE_CUDA(cudaEventRecord(hs->copied[b], ctx->copy_stream));
    return BE_OK;
  };
  if (hs) {
    // buffer b serves the chunks b, b + 2, ..: sized for the largest of them
    size_t need[2] = {0, 0};
    const std::vector<int64_t>& cb = feed_sub.empty() ? cstart : feed_sub;
    for (size_t ci = 0; ci + 1 < cb.size(); ++ci) {
      const size_t nb = (size_t)(cb[ci + 1] - cb[ci]) * hs->loop_bytes;
      if (nb > need[ci & 1]) need[ci & 1] = nb;
    }
    for (int b = 0; b < 2; ++b) {
      if (need[b] <= ctx->stage_cap[b]) continue;
      BE_CUDA(cudaStreamSynchronize(ctx->stream));
      if (ctx->stage_buf[b]) cudaFree(ctx->stage_buf[b]);
      ctx->stage_buf[b] = nullptr; ctx->stage_cap[b] = 0;
      if (cudaMalloc(&ctx->stage_buf[b], need[b]) != cudaSuccess) { cudaGetLastError(); return BE_ERR_NOMEM; }
      ctx->stage_cap[b] = need[b];
    }
    hs->stage[0] = ctx->stage_buf[0]; hs->stage[1] = ctx->stage_buf[1];
    memset(&smap, 0, sizeof(smap));
    smap.ndim = 1; smap.dir = 0; smap.n1 = n1; smap.dims[0] = n1; smap.stride[0] = 1; smap.batch_stride = n1; smap.loops = lc;
    BE_TRY(issue_copy(0));
    if (!feed_sub.empty()) BE_TRY(issue_copy(1));
  }
  HostFeed feed;
  if (hs) ctx->host_schedule = feed_sub.empty() ? (int)nchunks : -((int)feed_sub.size() - 1);
  if (!feed_sub.empty()) {
    feed.nsub = (int)feed_sub.size() - 1;
    for (size_t i = 0; i < feed_sub.size(); ++i) feed.mstart[i] = feed_sub[i] * n1;
    for (int b = 0; b < 2; ++b) { feed.buf[b] = hs->stage[b]; feed.copied[b] = hs->copied[b]; feed.freed[b] = hs->freed[b]; }
    feed.issue = [](void* self, int j) -> int { return (*(decltype(issue_copy)*)self)((int64_t)j); };
    feed.self = &issue_copy;
  }
  if (pipe) {
    BE_TRY(pipeline_init(ctx));
    if (be_arena_reserve(ctx, 2 * region + persist + (4 << 20)) != BE_OK) pipe = false;   // not enough memory: serial
  }
  if (!pipe) BE_TRY(be_arena_reserve(ctx, region + persist + (4 << 20)));
  cudaStream_t S1 = ctx->stream;
  cplx* Wall[2] = {nullptr, nullptr};
  // equal sectors: one contiguous buffer, so that both sectors' Wilson matrices are solved in ONE batch
  const bool joint = sp && msec[0] == msec[1] && msec[0] > 0 && sp->theta_lo && sp->theta_hi;
  if (joint) {
    Wall[0] = (cplx*)be_arena_alloc(ctx, 2 * (size_t)loops * msec[0] * msec[0] * sizeof(cplx));
    if (!Wall[0]) return BE_ERR_NOMEM;
    Wall[1] = Wall[0] + (size_t)loops * msec[0] * msec[0];
  } else {
    for (int s = 0; s < 2; ++s)
      if (msec[s] > 0) {
        Wall[s] = (cplx*)be_arena_alloc(ctx, (size_t)loops * msec[s] * msec[s] * sizeof(cplx));
        if (!Wall[s]) return BE_ERR_NOMEM;
      }
  }
  int* bad = (int*)be_arena_alloc(ctx, 2 * (size_t)loops * sizeof(int));
  if (!bad) return BE_ERR_NOMEM;
  BE_CUDA(cudaMemsetAsync(bad, 0, 2 * (size_t)loops * sizeof(int), ctx->stream));
  if (sp && sp->S_is_diag && N >= 64) {
    int* d_sel = (int*)be_arena_alloc(ctx, (size_t)N * sizeof(int));
    if (!d_sel) return BE_ERR_NOMEM;
    BE_TRY(analyze_diag_S(ctx, &spl, N, d_sel));
  }
  const size_t keep = ctx->arena_used;
  for (int64_t ci = 0; ci < nchunks; ++ci) {
    const int64_t l0 = cstart[ci], nl = cstart[ci + 1] - l0;
    const int64_t cnt = nl * n1;
    ctx->arena_used = keep + (pipe ? (size_t)(ci & 1) * region : 0);
    if (pipe) {
      ctx->stream = S1;
      if (ci >= 2) BE_CUDA(cudaStreamWaitEvent(S1, ctx->ev_region[ci & 1], 0));   // region free again
      ctx->split_after_tridiag = 1;
      ctx->gemm_pad = (ci + 1 < nchunks && N > 8) ? 1 : 0;   // a next chunk will stream its matrices next to these GEMMs
    }
    const cplx* Hc = H;
    if (hs && feed_sub.empty()) {
      if (ci + 1 < nchunks) BE_TRY(issue_copy(ci + 1));
      BE_CUDA(cudaStreamWaitEvent(ctx->stream, hs->copied[ci & 1], 0));
      Hc = (const cplx*)hs->stage[ci & 1];
    }
    ctx->bloch = bs;   // consumed (and cleared) by the H eigensolve of the chunk
    ctx->feed = feed_sub.empty() ? nullptr : &feed;   // likewise: the sub-ranges are gathered as they land
    const int rc = wilson_chunk(ctx, Hc, hs ? smap : map, hs ? 0 : l0, N, m, n1, l0, nl, cnt, d_close, d_mingap, sp, mlo,
                                mhi, Wall, bad, loops);
    ctx->bloch = nullptr;
    ctx->feed = nullptr;
    if (hs && feed_sub.empty() && rc == BE_OK) cudaEventRecord(hs->freed[ci & 1], ctx->stream);
    if (pipe) {
      ctx->split_after_tridiag = 0;
      if (rc == BE_OK) cudaEventRecord(ctx->ev_region[ci & 1], ctx->stream);
    }
    if (rc != BE_OK) { ctx->stream = S1; ctx->gemm_pad = 0; return rc; }
  }
  // ---- S4 for every loop at once
  ctx->arena_used = keep;
  int rc = BE_OK;
  if (!sp) {
    rc = be_eigenphases(ctx, Wall[0], loops, m, d_theta, d_abs, bad);
  } else if (joint) {
    // the solve is latency bound per matrix: 2 x loops matrices in one launch cost what loops do
    const size_t nb = (size_t)loops * msec[0] * sizeof(double);
    double* th = (double*)be_arena_alloc(ctx, 2 * nb);
    if (!th) rc = BE_ERR_NOMEM;
    if (rc == BE_OK) rc = be_eigenphases(ctx, Wall[0], 2 * loops, msec[0], th, nullptr, bad);
    if (rc == BE_OK) rc = (int)cudaMemcpyAsync(sp->theta_lo, th, nb, cudaMemcpyDeviceToDevice, ctx->stream);
    if (rc == BE_OK) rc = (int)cudaMemcpyAsync(sp->theta_hi, (char*)th + nb, nb, cudaMemcpyDeviceToDevice, ctx->stream);
  } else {
    for (int sector = 0; sector < 2 && rc == BE_OK; ++sector) {
      double* out = sector == 0 ? sp->theta_lo : sp->theta_hi;
      if (msec[sector] == 0 || !out) continue;
      rc = be_eigenphases(ctx, Wall[sector], loops, msec[sector], out, nullptr, bad + sector * loops);
    }
  }
  if (pipe) {   // join: the caller's stream waits for everything enqueued on stream2
    cudaEventRecord(ctx->ev_join, ctx->stream);
    cudaStreamWaitEvent(S1, ctx->ev_join, 0);
    ctx->stream = S1;
    ctx->gemm_pad = 0;
  }
  return rc;
}

// One chunk of nl whole loops (cnt = nl * n1 matrices): S1, then S6 (if sp), S2, S3 into Wall.
// gl0: first loop of the chunk inside (H, map); l0: first loop of the chunk in the outputs.
static int wilson_chunk(be_ctx* ctx, const cplx* H, const GridMap& map, int64_t gl0, int N, int m, int n1, int64_t l0,
                        int64_t nl, int64_t cnt, const cplx* d_close, double* d_mingap, const SpinArgs* sp, int mlo,
                        int mhi, cplx* const* Wall, int* bad, int64_t loops) {
  {
    const int lo = ctx->band_lo, hi = lo + m;   // band window [lo, hi): the lowest hi vectors are computed
    double* E = (double*)be_arena_alloc(ctx, (size_t)cnt * N * sizeof(double));
    cplx* X = (cplx*)be_arena_alloc(ctx, (size_t)cnt * N * hi * sizeof(cplx));
    int* info = (int*)be_arena_alloc(ctx, (size_t)cnt * sizeof(int));
    if (!E || !X || !info) return BE_ERR_NOMEM;
    {
      const int r = be_eigh_frames(ctx, H, map, gl0, cnt, N, hi, hi + 1, E, X, info);
      ctx->bloch = nullptr;   // only H(k) is generated; the PSO solve below reads S_red from memory
      BE_TRY(r);
    }
    // loops with a flagged eigensolve get NaN phases at the end (bad[0 .. loops) lower / plain, [loops ..) upper)
    BE_TRY(be_flag_loops(ctx, info, E, N, n1, nl, bad + l0, sp ? bad + loops + l0 : nullptr));
    if (d_mingap) BE_TRY(be_mingap(ctx, E, N, lo, hi, n1, nl, d_mingap + l0));
    if (lo > 0) {
      // frames are column-major N x hi per k-point: columns lo .. hi-1 are one contiguous run per frame
      cplx* F = (cplx*)be_arena_alloc(ctx, (size_t)cnt * N * m * sizeof(cplx));
      if (!F) return BE_ERR_NOMEM;
      BE_CUDA(cudaMemcpy2DAsync(F, (size_t)N * m * sizeof(cplx), X + (size_t)lo * N, (size_t)N * hi * sizeof(cplx),
                                (size_t)N * m * sizeof(cplx), (size_t)cnt, cudaMemcpyDeviceToDevice, ctx->stream));
      X = F;
    }
    if (!sp) {
      cplx* W = nullptr;
      BE_TRY(be_chain_product(ctx, X, N, m, nl, n1, d_close, n1 - 1, Wall[0] + l0 * (int64_t)m * m, &W));
      return BE_OK;
    }
    cplx* V = nullptr;
    double* sig = nullptr;
    BE_TRY(pso_eigenvectors(ctx, X, cnt, N, m, sp, sp->pso ? sp->pso + l0 * (int64_t)n1 * m : nullptr, &V, info, &sig));
    BE_TRY(be_flag_loops(ctx, info, sig, m, n1, nl, bad + l0, bad + loops + l0));
    for (int sector = 0; sector < 2; ++sector) {
      const int ms = sector == 0 ? mlo : mhi;
      double* out = sector == 0 ? sp->theta_lo : sp->theta_hi;
      if (ms == 0 || !out) continue;
      const size_t mark = ctx->arena_used;
      cplx* F = (cplx*)be_arena_alloc(ctx, (size_t)cnt * N * ms * sizeof(cplx));
      if (!F) return BE_ERR_NOMEM;
      ZgemmParams g = zgemm_simple(N, ms, m, X, N, (int64_t)N * m, V + (sector ? (int64_t)mlo * m : 0), m,
                                   (int64_t)m * m, F, N, (int64_t)N * ms, cnt);
      BE_TRY(be_zgemm(ctx, BE_OP_N, BE_OP_N, g));
      cplx* W = nullptr;
      BE_TRY(be_chain_product(ctx, F, N, ms, nl, n1, d_close, n1 - 1, Wall[sector] + l0 * (int64_t)ms * ms, &W));
      ctx->arena_used = mark;
    }
  }
  return BE_OK;
}

size_t be_wilson_per_loop_bytes(int N, int m, int n1, int spin) { return per_loop_bytes(N, m, n1, spin != 0); }

static int check_common(be_ctx* ctx, const void* H, const be_grid* g, int n_occ, int dir) {
  if (!ctx || !H || !g) return BE_ERR_NULL;
  if (g->ndim < 1 || g->ndim > 3 || g->batch < 1 || g->N < 1) return BE_ERR_SHAPE;
  if (dir < 0 || dir >= g->ndim) return BE_ERR_SHAPE;
  if (n_occ < 1 || n_occ > g->N) return BE_ERR_SHAPE;
  if (!aligned(H, 16)) return BE_ERR_ALIGN;
  // size limits of the kernels, checked before anything is enqueued: the blocked eigensolver keeps two vectors of
  // length N in shared memory (N <= 6400), the QR iteration of the Wilson matrix owns columns in registers (m <= 2048)
  if (g->N > BE_MAX_N || n_occ > BE_MAX_M) return BE_ERR_UNSUPPORTED;
  return BE_OK;
}

extern "C" int be_wilson_loop(be_ctx* ctx, const void* dH_grid, const be_grid* grid, int n_occ, int dir,
                              const void* d_close, double* d_theta, double* d_abs, double* d_mingap) {
  BE_DEVICE_GUARD(ctx);
  BE_TRY(check_common(ctx, dH_grid, grid, n_occ, dir));
  if (!d_theta) return BE_ERR_NULL;
  if ((d_close && !aligned(d_close, 16)) || !aligned(d_theta, 8)) return BE_ERR_ALIGN;
  GridMap map;
  BE_TRY(make_map(grid, dir, &map));
  return wilson_device(ctx, (const cplx*)dH_grid, map, grid->N, n_occ, (const cplx*)d_close,
                       d_theta, d_abs, d_mingap, nullptr);
}

extern "C" int be_wilson_loop_window(be_ctx* ctx, const void* dH_grid, const be_grid* grid, int band_lo, int band_hi,
                                     int dir, const void* d_close, double* d_theta, double* d_abs, double* d_mingap) {
  BE_DEVICE_GUARD(ctx);
  if (band_lo < 0 || band_hi <= band_lo) return BE_ERR_SHAPE;
  BE_TRY(check_common(ctx, dH_grid, grid, band_hi, dir));
  if (!d_theta) return BE_ERR_NULL;
  if ((d_close && !aligned(d_close, 16)) || !aligned(d_theta, 8)) return BE_ERR_ALIGN;
  GridMap map;
  BE_TRY(make_map(grid, dir, &map));
  ctx->band_lo = band_lo;
  const int rc = wilson_device(ctx, (const cplx*)dH_grid, map, grid->N, band_hi - band_lo, (const cplx*)d_close,
                               d_theta, d_abs, d_mingap, nullptr);
  ctx->band_lo = 0;
  return rc;
}

extern "C" int be_spin_resolved_wilson_window(be_ctx* ctx, const void* dH_grid, const be_grid* grid, int band_lo,
                                              int band_hi, int dir, const void* dS, int S_is_diag, int m_lo,
                                              const void* d_close, double* d_theta_lo, double* d_theta_hi,
                                              double* d_pso) {
  BE_DEVICE_GUARD(ctx);
  if (band_lo < 0 || band_hi <= band_lo) return BE_ERR_SHAPE;
  BE_TRY(check_common(ctx, dH_grid, grid, band_hi, dir));
  if (!dS) return BE_ERR_NULL;
  const int m = band_hi - band_lo;
  if (m_lo < 0) m_lo = m / 2;
  if (m_lo > m) return BE_ERR_SHAPE;
  if (!aligned(dS, S_is_diag ? 8 : 16) || (d_close && !aligned(d_close, 16))) return BE_ERR_ALIGN;
  GridMap map;
  BE_TRY(make_map(grid, dir, &map));
  SpinArgs sp{dS, S_is_diag, m_lo, d_theta_lo, d_theta_hi, d_pso};
  ctx->band_lo = band_lo;
  const int rc = wilson_device(ctx, (const cplx*)dH_grid, map, grid->N, m, (const cplx*)d_close,
                               nullptr, nullptr, nullptr, &sp);
  ctx->band_lo = 0;
  return rc;
}

extern "C" int be_spin_resolved_wilson(be_ctx* ctx, const void* dH_grid, const be_grid* grid, int n_occ,
                                       int dir, const void* dS, int S_is_diag, int m_lo,
                                       const void* d_close, double* d_theta_lo, double* d_theta_hi,
                                       double* d_pso) {
  BE_DEVICE_GUARD(ctx);
  BE_TRY(check_common(ctx, dH_grid, grid, n_occ, dir));
  if (!dS) return BE_ERR_NULL;
  if (m_lo < 0) m_lo = n_occ / 2;
  if (m_lo > n_occ) return BE_ERR_SHAPE;
  if (!aligned(dS, S_is_diag ? 8 : 16) || (d_close && !aligned(d_close, 16))) return BE_ERR_ALIGN;
  GridMap map;
  BE_TRY(make_map(grid, dir, &map));
  SpinArgs sp{dS, S_is_diag, m_lo, d_theta_lo, d_theta_hi, d_pso};
  return wilson_device(ctx, (const cplx*)dH_grid, map, grid->N, n_occ, (const cplx*)d_close,
                       nullptr, nullptr, nullptr, &sp);
}

// ---------------------------------------------------------------------------------------------
extern "C" int be_nested_wilson(be_ctx* ctx, const void* dH_grid, const be_grid* grid, int n_occ,
                                int dir1, int dir2, int base, int wb_lo, int wb_hi, double theta_cut,
                                const void* d_close1, const void* d_close2,
                                double* d_theta1, double* d_theta_nested) {
  BE_DEVICE_GUARD(ctx);
  BE_TRY(check_common(ctx, dH_grid, grid, n_occ, dir1));
  be_subspace_guard subspace(ctx);
  if (!d_theta_nested) return BE_ERR_NULL;
  if (grid->ndim < 2 || dir2 < 0 || dir2 >= grid->ndim || dir2 == dir1) return BE_ERR_SHAPE;
  if (base < 0 || base >= grid->dims[dir1]) return BE_ERR_SHAPE;
  if (wb_lo < 0 || wb_hi > n_occ || wb_lo >= wb_hi) return BE_ERR_SHAPE;
  if (n_occ > 2 && wb_hi - wb_lo > 64) return BE_ERR_UNSUPPORTED;   // inverse-iteration path: at most 64 Wannier bands (header)
  const int N = grid->N, m = n_occ, ns = wb_hi - wb_lo;
  // virtual axis order (other, dir2, dir1) so that loops enumerate [batch][other][i2]
  GridMap full;
  BE_TRY(make_map(grid, dir1, &full));
  GridMap map;
  memset(&map, 0, sizeof(map));
  int other = -1;
  for (int a = 0; a < grid->ndim; ++a) if (a != dir1 && a != dir2) other = a;
  int k = 0;
  if (other >= 0) { map.dims[k] = full.dims[other]; map.stride[k] = full.stride[other]; ++k; }
  map.dims[k] = full.dims[dir2]; map.stride[k] = full.stride[dir2]; ++k;
  map.dims[k] = full.dims[dir1]; map.stride[k] = full.stride[dir1];
  map.ndim = k + 1; map.dir = k; map.n1 = full.n1; map.shift = base;
  map.batch_stride = full.batch_stride; map.loops = full.loops;
  const int n1 = map.n1, n2 = grid->dims[dir2];
  const int64_t loops = map.loops, outer2 = loops / n2;
  const int phi_at = n1 - 1 - base;   // link whose target frame has grid index 0

  const size_t per = (size_t)n1 * (be_eigh_scratch_bytes(1, N, m) + (size_t)N * m * 16 + (size_t)N * 8 + 512)
                     + (size_t)2 * n1 * m * m * 16 + 8 * (size_t)m * m * 16 + 4096
                     + (m > 2 ? be_nested_general_scratch_bytes(1, m, ns) + be_eigenphases_scratch_bytes(1, m) : 0);
  const size_t persist = (size_t)loops * ((size_t)N * ns * 16 + 256) + (size_t)outer2 * (2 * n2 + 8) * ns * ns * 16 + (8 << 20);
  int64_t lc = (int64_t)(be_effective_ws_limit(ctx, per * (size_t)loops) / per);
  if (lc < 1) lc = 1;
  if (lc > loops) lc = loops;
  BE_TRY(be_arena_reserve(ctx, per * (size_t)lc + persist + (size_t)loops * m * 8 + (4 << 20)));
  // persistent across chunks: Wannier-band frames and (optional) first-level phases
  cplx* Wf = (cplx*)be_arena_alloc(ctx, (size_t)loops * N * ns * sizeof(cplx));
  double* th1 = d_theta1 ? d_theta1 : (double*)be_arena_alloc(ctx, (size_t)loops * m * sizeof(double));
  if (!Wf || !th1) return BE_ERR_NOMEM;
  const size_t keep = ctx->arena_used;
  const bool fused = be_small_loop_applies(N, m, n1);
  if (fused) {
    // first level in one kernel: W of every loop and the frame at the base point, nothing else is written
    cplx* W = (cplx*)be_arena_alloc(ctx, (size_t)loops * m * m * sizeof(cplx));
    cplx* X0 = (cplx*)be_arena_alloc(ctx, (size_t)loops * N * m * sizeof(cplx));
    cplx* Vs = (cplx*)be_arena_alloc(ctx, (size_t)loops * m * ns * sizeof(cplx));
    if (!W || !X0 || !Vs) return BE_ERR_NOMEM;
    BE_TRY(be_small_loop(ctx, (const cplx*)dH_grid, nullptr, map, N, m, (const cplx*)d_close1, phi_at, nullptr, nullptr, nullptr, W, X0,
                         nullptr, 0, 0, nullptr, nullptr, nullptr));
    BE_TRY(be_nested_select_small(ctx, W, loops, m, wb_lo, wb_hi, theta_cut, th1, Vs));
    ZgemmParams g = zgemm_simple(N, ns, m, X0, N, (int64_t)N * m, Vs, m, (int64_t)m * ns, Wf, N, (int64_t)N * ns, loops);
    BE_TRY(be_zgemm(ctx, BE_OP_N, BE_OP_N, g));
  }
  for (int64_t l0 = 0; l0 < loops && !fused; l0 += lc) {
    const int64_t nl = (loops - l0 < lc) ? loops - l0 : lc;
    const int64_t cnt = nl * n1;
    ctx->arena_used = keep;
    double* E = (double*)be_arena_alloc(ctx, (size_t)cnt * N * sizeof(double));
    cplx* X = (cplx*)be_arena_alloc(ctx, (size_t)cnt * N * m * sizeof(cplx));
    cplx* Vs = (cplx*)be_arena_alloc(ctx, (size_t)nl * m * ns * sizeof(cplx));
    if (!E || !X || !Vs) return BE_ERR_NOMEM;
    BE_TRY(be_eigh_frames(ctx, (const cplx*)dH_grid, map, l0, cnt, N, m, m + 1, E, X, nullptr));
    cplx* W = nullptr;
    BE_TRY(be_chain_product(ctx, X, N, m, nl, n1, (const cplx*)d_close1, phi_at, nullptr, &W));
    if (m <= 2) BE_TRY(be_nested_select_small(ctx, W, nl, m, wb_lo, wb_hi, theta_cut, th1 + l0 * m, Vs));
    else BE_TRY(be_nested_select_general(ctx, W, nl, m, wb_lo, wb_hi, theta_cut, th1 + l0 * m, Vs));
    // w = U_base V_S  (frame j = 0 of each rolled loop)
    ZgemmParams g = zgemm_simple(N, ns, m, X, N, (int64_t)n1 * N * m, Vs, m, (int64_t)m * ns,
                                 Wf + l0 * (int64_t)N * ns, N, (int64_t)N * ns, nl);
    BE_TRY(be_zgemm(ctx, BE_OP_N, BE_OP_N, g));
  }
  ctx->arena_used = keep;
  if (be_small_loop_applies(N, ns, n2)) {
    // second level on the Wannier-band frames in one kernel as well
    GridMap m2;
    memset(&m2, 0, sizeof(m2));
    m2.ndim = 1; m2.dir = 0; m2.n1 = n2; m2.dims[0] = n2; m2.stride[0] = 1; m2.batch_stride = n2; m2.loops = outer2;
    return be_small_loop(ctx, nullptr, Wf, m2, N, ns, (const cplx*)d_close2, n2 - 1, d_theta_nested, nullptr, nullptr, nullptr,
                         nullptr, nullptr, 0, 0, nullptr, nullptr, nullptr);
  }
  cplx* W2 = nullptr;
  BE_TRY(be_chain_product(ctx, Wf, N, ns, outer2, n2, (const cplx*)d_close2, n2 - 1, nullptr, &W2));
  BE_TRY(be_eigenphases(ctx, W2, outer2, ns, d_theta_nested, nullptr));
  return BE_OK;
}

// ---------------------------------------------------------------------------------------------
// NEXT-2: plaquette Berry fluxes on a periodic 2D grid (include/berryeasy_b200.h)
static ZgemmParams link_params(const cplx* A, const cplx* B, cplx* C, int M, int Nn, int K, int lda, int ldb,
                               int64_t sAi, int64_t sAo, int64_t sBi, int64_t sBo, int64_t sCi, int64_t sCo,
                               int inner, int64_t batch, int ring) {
  ZgemmParams g = zgemm_simple(M, Nn, K, A, lda, sAo, B, ldb, sBo, C, M, sCo, batch);
  g.sAi = sAi; g.sBi = sBi; g.sCi = sCi; g.inner = inner; g.ringB = ring; g.phi_at = -1;
  return g;
}

// fluxes of one set of frames F [batch][ny][nx][ms][N]
static int plaquette_of_frames(be_ctx* ctx, const cplx* F, int64_t batch, int ny, int nx, int N, int ms,
                               double* d_flux) {
  const int64_t pts = (int64_t)ny * nx, mm = (int64_t)ms * ms, fr = (int64_t)N * ms;
  cplx* Lx = (cplx*)be_arena_alloc(ctx, (size_t)batch * pts * mm * sizeof(cplx));
  cplx* Ly = (cplx*)be_arena_alloc(ctx, (size_t)batch * pts * mm * sizeof(cplx));
  cplx* P1 = (cplx*)be_arena_alloc(ctx, (size_t)batch * pts * mm * sizeof(cplx));
  cplx* P2 = (cplx*)be_arena_alloc(ctx, (size_t)batch * pts * mm * sizeof(cplx));
  if (!Lx || !Ly || !P1 || !P2) return BE_ERR_NOMEM;
  for (int64_t bt = 0; bt < batch; ++bt) {
    const cplx* Fb = F + bt * pts * fr;
    cplx *lx = Lx + bt * pts * mm, *ly = Ly + bt * pts * mm, *p1 = P1 + bt * pts * mm, *p2 = P2 + bt * pts * mm;
    // L_x(j,i) = F(j,i)^H F(j,i+1): ring over i inside every row j
    BE_TRY(be_zgemm(ctx, BE_OP_C, BE_OP_N, link_params(Fb, Fb, lx, ms, ms, N, N, N, fr, nx * fr, fr, nx * fr, mm, nx * mm, nx, pts, 1)));
    // L_y(j,i) = F(j,i)^H F(j+1,i): ring over j inside every column i (stored [j][i] like L_x)
    BE_TRY(be_zgemm(ctx, BE_OP_C, BE_OP_N, link_params(Fb, Fb, ly, ms, ms, N, N, N, nx * fr, fr, nx * fr, fr, nx * mm, mm, ny, pts, 1)));
    // P1(j,i) = L_x(j,i) L_y(j,i+1)
    BE_TRY(be_zgemm(ctx, BE_OP_N, BE_OP_N, link_params(lx, ly, p1, ms, ms, ms, ms, ms, mm, nx * mm, mm, nx * mm, mm, nx * mm, nx, pts, 1)));
    // P2(j,i) = P1(j,i) L_x(j+1,i)^H
    BE_TRY(be_zgemm(ctx, BE_OP_N, BE_OP_C, link_params(p1, lx, p2, ms, ms, ms, ms, ms, nx * mm, mm, nx * mm, mm, nx * mm, mm, ny, pts, 1)));
    // P1 <- P2(j,i) L_y(j,i)^H: the closed loop around the plaquette
    BE_TRY(be_zgemm(ctx, BE_OP_N, BE_OP_C, link_params(p2, ly, p1, ms, ms, ms, ms, ms, mm, nx * mm, mm, nx * mm, mm, nx * mm, nx, pts, 0)));
  }
  return be_det_phase(ctx, P1, batch * pts, ms, d_flux);
}

extern "C" int be_plaquette_flux(be_ctx* ctx, const void* dH_grid, const be_grid* grid, int n_occ, const void* dS,
                                 int S_is_diag, int m_lo, double* d_flux, double* d_flux_hi, double* d_pso) {
  BE_DEVICE_GUARD(ctx);
  BE_TRY(check_common(ctx, dH_grid, grid, n_occ, 0));
  be_subspace_guard subspace(ctx);
  if (grid->ndim != 2 || !d_flux) return grid->ndim != 2 ? BE_ERR_SHAPE : BE_ERR_NULL;
  const int ny = grid->dims[0], nx = grid->dims[1], N = grid->N, m = n_occ;
  if (dS) {
    if (m_lo < 0) m_lo = m / 2;
    if (m_lo > m || !aligned(dS, S_is_diag ? 8 : 16)) return m_lo > m ? BE_ERR_SHAPE : BE_ERR_ALIGN;
  }
  GridMap map;
  BE_TRY(make_map(grid, 1, &map));           // points enumerated [batch][ny][nx]
  const int64_t cnt = grid->batch * ny * nx;
  // everything of the grid is live at once (every point is a corner of four plaquettes)
  const size_t mmax = (size_t)m * m * sizeof(cplx);
  const size_t need = (size_t)cnt * (be_eigh_scratch_bytes(1, N, m) + 2 * (size_t)N * m * sizeof(cplx) + N * sizeof(double) +
                                     (dS ? (size_t)N * m * sizeof(cplx) + 3 * mmax + be_eigh_scratch_bytes(1, m, m) : 0) +
                                     6 * mmax + 4096) + (8 << 20);
  if (need > be_effective_ws_limit(ctx, need)) return BE_ERR_UNSUPPORTED;   // the grid has to fit one chunk (header)
  BE_TRY(be_arena_reserve(ctx, need));
  double* E = (double*)be_arena_alloc(ctx, (size_t)cnt * N * sizeof(double));
  cplx* X = (cplx*)be_arena_alloc(ctx, (size_t)cnt * N * m * sizeof(cplx));
  if (!E || !X) return BE_ERR_NOMEM;
  BE_TRY(be_eigh_frames(ctx, (const cplx*)dH_grid, map, 0, cnt, N, m, m + 1, E, X, nullptr));
  if (!dS) return plaquette_of_frames(ctx, X, grid->batch, ny, nx, N, m, d_flux);
  SpinArgs sp{dS, S_is_diag, m_lo, nullptr, nullptr, d_pso};
  cplx* V = nullptr;
  BE_TRY(pso_eigenvectors(ctx, X, cnt, N, m, &sp, d_pso, &V, nullptr, nullptr));
  const int msz[2] = {m_lo, m - m_lo};
  double* outs[2] = {d_flux, d_flux_hi};
  for (int sector = 0; sector < 2; ++sector) {
    const int ms = msz[sector];
    if (ms == 0 || !outs[sector]) continue;
    const size_t mark = ctx->arena_used;
    cplx* F = (cplx*)be_arena_alloc(ctx, (size_t)cnt * N * ms * sizeof(cplx));
    if (!F) return BE_ERR_NOMEM;
    ZgemmParams g = zgemm_simple(N, ms, m, X, N, (int64_t)N * m, V + (sector ? (int64_t)m_lo * m : 0), m,
                                 (int64_t)m * m, F, N, (int64_t)N * ms, cnt);
    BE_TRY(be_zgemm(ctx, BE_OP_N, BE_OP_N, g));
    BE_TRY(plaquette_of_frames(ctx, F, grid->batch, ny, nx, N, ms, outs[sector]));
    ctx->arena_used = mark;
  }
  return BE_OK;
}

// host-resident grid (api_host.cu): same chunking, deferred eigenphases and scratch as the device path
int be_wilson_host_device(be_ctx* ctx, HostStage* hs, const be_grid* grid, int dir, int m, const void* d_close,
                          double* d_theta, double* d_abs, double* d_mingap, const void* dS, int S_is_diag, int m_lo,
                          double* d_theta_lo, double* d_theta_hi, double* d_pso, int spin) {
  BE_TRY(make_map(grid, dir, &hs->hmap));
  const int n1 = hs->hmap.n1, N = grid->N;
  const int64_t loops = hs->hmap.loops;
  // inside a staged chunk the loops are contiguous whatever the direction in the host grid was
  GridMap map;
  memset(&map, 0, sizeof(map));
  map.ndim = 1; map.dir = 0; map.n1 = n1; map.dims[0] = n1; map.stride[0] = 1; map.batch_stride = n1; map.loops = loops;
  if (!spin) return wilson_device(ctx, nullptr, map, N, m, (const cplx*)d_close, d_theta, d_abs, d_mingap, nullptr, hs);
  SpinArgs sp{dS, S_is_diag, m_lo, d_theta_lo, d_theta_hi, d_pso};
  return wilson_device(ctx, nullptr, map, N, m, (const cplx*)d_close, nullptr, nullptr, nullptr, &sp, hs);
}

// ---------------------------------------------------------------------------------------------
// NEXT-1 fused in front of S1: the loops of a grid whose H(k) is generated chunk by chunk from real-space
// blocks (no H_grid in memory).
static int bloch_source(be_ctx* ctx, const void* dA, const int* h_R, int nR, const be_grid* grid, int dir,
                        BlochSrc* bs) {
  if (!dA || !h_R) return BE_ERR_NULL;
  if (nR < 1) return BE_ERR_SHAPE;
  if (!aligned(dA, 16)) return BE_ERR_ALIGN;
  BE_TRY(make_map(grid, dir, &bs->map));
  const size_t need = (size_t)nR * grid->ndim * sizeof(int);
  if (need > ctx->dR_cap) {
    if (ctx->dR_buf) { BE_CUDA(cudaStreamSynchronize(ctx->stream)); cudaFree(ctx->dR_buf); ctx->dR_buf = nullptr; ctx->dR_cap = 0; }
    if (cudaMalloc((void**)&ctx->dR_buf, need) != cudaSuccess) { cudaGetLastError(); return BE_ERR_NOMEM; }
    ctx->dR_cap = need;
  }
  BE_CUDA(cudaMemcpyAsync(ctx->dR_buf, h_R, need, cudaMemcpyHostToDevice, ctx->stream));
  bs->A = (const cplx*)dA; bs->dR = ctx->dR_buf; bs->nR = nR;
  bs->loops_per_batch = bs->map.loops / grid->batch;
  return BE_OK;
}

extern "C" int be_wilson_loop_bloch(be_ctx* ctx, const void* dA, const int* h_R, int nR, const be_grid* grid,
                                    int n_occ, int dir, const void* d_close, double* d_theta, double* d_abs,
                                    double* d_mingap) {
  BE_DEVICE_GUARD(ctx);
  BE_TRY(check_common(ctx, dA, grid, n_occ, dir));
  if (!d_theta) return BE_ERR_NULL;
  BlochSrc bs;
  BE_TRY(bloch_source(ctx, dA, h_R, nR, grid, dir, &bs));
  return wilson_device(ctx, nullptr, bs.map, grid->N, n_occ, (const cplx*)d_close, d_theta, d_abs, d_mingap, nullptr,
                       nullptr, &bs);
}

extern "C" int be_spin_resolved_wilson_bloch(be_ctx* ctx, const void* dA, const int* h_R, int nR, const be_grid* grid,
                                             int n_occ, int dir, const void* dS, int S_is_diag, int m_lo,
                                             const void* d_close, double* d_theta_lo, double* d_theta_hi,
                                             double* d_pso) {
  BE_DEVICE_GUARD(ctx);
  BE_TRY(check_common(ctx, dA, grid, n_occ, dir));
  if (!dS) return BE_ERR_NULL;
  if (m_lo < 0) m_lo = n_occ / 2;
  if (m_lo > n_occ) return BE_ERR_SHAPE;
  BlochSrc bs;
  BE_TRY(bloch_source(ctx, dA, h_R, nR, grid, dir, &bs));
  SpinArgs sp{dS, S_is_diag, m_lo, d_theta_lo, d_theta_hi, d_pso};
  return wilson_device(ctx, nullptr, bs.map, grid->N, n_occ, (const cplx*)d_close, nullptr, nullptr, nullptr, &sp,
                       nullptr, &bs);
}
