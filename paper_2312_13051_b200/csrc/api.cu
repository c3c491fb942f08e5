// C-ABI entry points (include/berryeasy_b200.h): argument checks, scratch arena, chunking over
// whole loops, sequencing of the stages.  All arithmetic is in the kernels of the other files.
#include "be_common.cuh"
#include <new>
#include <vector>
#include <string.h>

// stage entry points defined in wilson.cu
int be_mingap(be_ctx* ctx, const double* E, int N, int lo, int hi, int n1, int64_t loops, double* out);
int be_scale_rows(be_ctx* ctx, const cplx* X, const double* S, cplx* SX, int N, int64_t total);
int be_winding_impl(be_ctx* ctx, const double* theta, int64_t n_cycles, int n_points, int m, double* wind);
int be_nested_select_small(be_ctx* ctx, const cplx* W, int64_t cnt, int m, int wb_lo, int wb_hi,
                           double cut, double* theta1, cplx* Vs);
int be_chain_product(be_ctx* ctx, const cplx* F, int N, int m, int64_t outer, int n1,
                     const cplx* d_close, int phi_at, cplx* Wdst, cplx** Wout);

// ---------------------------------------------------------------------------------------------
// optional profile: one CUDA event pair per launch of the instrumented kernel classes
struct be_prof {
  bool on = false;
  std::vector<cudaEvent_t> ev;     // pairs
  std::vector<int> cls;
  size_t used = 0;                 // pairs in use
  double bytes[PK_COUNT] = {0}, flops[PK_COUNT] = {0};
  int64_t count[PK_COUNT] = {0};
};

void be_prof_begin(be_ctx* ctx, int cls) {
  be_prof* p = ctx->prof;
  if (!p || !p->on) return;
  if (p->used * 2 >= p->ev.size()) {
    for (int i = 0; i < 2048; ++i) { cudaEvent_t e; cudaEventCreate(&e); p->ev.push_back(e); }
    p->cls.resize(p->ev.size() / 2);
  }
  p->cls[p->used] = cls;
  cudaEventRecord(p->ev[2 * p->used], ctx->stream);
}

void be_prof_end(be_ctx* ctx, int cls, double bytes, double flops) {
  be_prof* p = ctx->prof;
  if (!p || !p->on) return;
  cudaEventRecord(p->ev[2 * p->used + 1], ctx->stream);
  p->used++;
  p->bytes[cls] += bytes; p->flops[cls] += flops; p->count[cls]++;
}

extern "C" int be_profile_enable(be_ctx* ctx, int on) {
  BE_DEVICE_GUARD(ctx);
  if (!ctx) return BE_ERR_NULL;
  if (!ctx->prof) ctx->prof = new (std::nothrow) be_prof;
  if (!ctx->prof) return BE_ERR_NOMEM;
  be_prof* p = ctx->prof;
  BE_CUDA(cudaStreamSynchronize(ctx->stream));
  p->on = on != 0;
  p->used = 0;
  for (int i = 0; i < PK_COUNT; ++i) { p->bytes[i] = p->flops[i] = 0; p->count[i] = 0; }
  return BE_OK;
}

extern "C" const char* be_profile_name(int cls) {
  static const char* names[PK_COUNT] = {"hemv", "colw", "zgemm", "bisect", "invit", "cluster_orth",
                                        "hessenberg", "hqr", "jacobi", "misc", "fused", "panel", "chase", "q2"};
  return (cls >= 0 && cls < PK_COUNT) ? names[cls] : nullptr;
}

extern "C" int be_profile_get(be_ctx* ctx, int cls, double* ms, int64_t* launches, double* bytes, double* flops) {
  BE_DEVICE_GUARD(ctx);
  if (!ctx || !ctx->prof) return BE_ERR_NULL;
  if (cls < 0 || cls >= PK_COUNT) return BE_ERR_SHAPE;
  be_prof* p = ctx->prof;
  BE_CUDA(cudaStreamSynchronize(ctx->stream));
  double tot = 0;
  for (size_t i = 0; i < p->used; ++i)
    if (p->cls[i] == cls) { float t = 0; cudaEventElapsedTime(&t, p->ev[2 * i], p->ev[2 * i + 1]); tot += t; }
  if (ms) *ms = tot;
  if (launches) *launches = p->count[cls];
  if (bytes) *bytes = p->bytes[cls];
  if (flops) *flops = p->flops[cls];
  return BE_OK;
}

// ---------------------------------------------------------------------------------------------
// arena
int be_arena_reserve(be_ctx* ctx, size_t bytes) {
  ctx->arena_used = 0;
  if (bytes <= ctx->arena_bytes) return BE_OK;
  if (ctx->arena) {
    BE_CUDA(cudaStreamSynchronize(ctx->stream));
    BE_CUDA(cudaFree(ctx->arena));
    ctx->arena = nullptr; ctx->arena_bytes = 0;
  }
  void* p = nullptr;
  cudaError_t e = cudaMalloc(&p, bytes);
  if (e != cudaSuccess) { cudaGetLastError(); return BE_ERR_NOMEM; }
  ctx->arena = (char*)p; ctx->arena_bytes = bytes;
  return BE_OK;
}

// The cap that applies to a call: the configured limit, but never more than what the device can give right now
// (free memory plus the arena already held, minus a margin for the caller's outputs and the CUDA context).
// host_grid: the grid is not resident on the device, so the DEFAULT cap (70 % of the memory, which leaves room
// for a device-resident grid) is raised to 85 %; a cap set by the caller stands.
size_t be_effective_ws_limit(be_ctx* ctx, size_t want, bool host_grid) {
  size_t lim = ctx->ws_limit;
  if (host_grid && !ctx->ws_user) { const size_t l2 = (size_t)(0.85 * (double)ctx->total_mem); if (l2 > lim) lim = l2; }
  // cudaMemGetInfo costs ~0.5 ms: not worth asking when the whole request is small or already held
  if (want <= ctx->arena_bytes || want <= ((size_t)1 << 30)) return lim;
  size_t fr = 0, tot = 0;
  if (cudaMemGetInfo(&fr, &tot) != cudaSuccess) { cudaGetLastError(); return lim; }
  const size_t margin = (size_t)2 << 30;
  size_t avail = fr + ctx->arena_bytes;
  avail = avail > margin ? avail - margin : avail / 2;
  return lim < avail ? lim : avail;
}

void* be_arena_alloc(be_ctx* ctx, size_t bytes) {
  const size_t b = be_align256(bytes ? bytes : 1);
  if (ctx->arena_used + b > ctx->arena_bytes) return nullptr;
  void* p = ctx->arena + ctx->arena_used;
  ctx->arena_used += b;
  return p;
}

// ---------------------------------------------------------------------------------------------
extern "C" int be_create(be_ctx** out, void* cuda_stream) {
  if (!out) return BE_ERR_NULL;
  be_ctx* c = new (std::nothrow) be_ctx;
  if (!c) return BE_ERR_NOMEM;
  memset(c, 0, sizeof(*c));
  c->stream = (cudaStream_t)cuda_stream;
  cudaError_t e = cudaGetDevice(&c->device);
  if (e != cudaSuccess) { delete c; return (int)e; }
  cudaDeviceProp prop;
  e = cudaGetDeviceProperties(&prop, c->device);
  if (e != cudaSuccess) { delete c; return (int)e; }
  c->sm_count = prop.multiProcessorCount;
  // scratch cap: 70 % of the device memory (134 GB on a B200).  Larger chunks fill the one-CTA-per-matrix kernels'
  // waves better (600 matrices in one chunk instead of 2 x 300: 2481 vs 2561 ms on the bench workload)
  c->ws_limit = (size_t)(0.70 * (double)prop.totalGlobalMem);
  c->total_mem = prop.totalGlobalMem;
  c->ws_user = 0;
  if (c->ws_limit < ((size_t)4 << 30)) c->ws_limit = (size_t)4 << 30;
  c->eigh_algo = 2;
  c->invit_solves = 3;
  c->h2d_bytes = 0;
  *out = c;
  return BE_OK;
}

extern "C" int be_destroy(be_ctx* ctx) {
  BE_DEVICE_GUARD(ctx);
  if (!ctx) return BE_ERR_NULL;
  cudaStreamSynchronize(ctx->stream);
  if (ctx->arena) cudaFree(ctx->arena);
  if (ctx->copy_stream) cudaStreamDestroy(ctx->copy_stream);
  if (ctx->dR_buf) cudaFree(ctx->dR_buf);
  for (int i = 0; i < 2; ++i) if (ctx->stage_buf[i]) cudaFree(ctx->stage_buf[i]);
  if (ctx->stream2) {
    cudaStreamDestroy(ctx->stream2);
    cudaEventDestroy(ctx->ev_split); cudaEventDestroy(ctx->ev_join);
    cudaEventDestroy(ctx->ev_region[0]); cudaEventDestroy(ctx->ev_region[1]);
  }
  if (ctx->side_stream) { cudaStreamDestroy(ctx->side_stream); cudaEventDestroy(ctx->ev_side[0]); cudaEventDestroy(ctx->ev_side[1]); }
  if (ctx->prof) { for (cudaEvent_t e : ctx->prof->ev) cudaEventDestroy(e); delete ctx->prof; }
  delete ctx;
  return BE_OK;
}

extern "C" const char* be_strerror(int code) {
  switch (code) {
    case BE_OK: return "ok";
    case BE_ERR_NULL: return "required pointer is NULL";
    case BE_ERR_SHAPE: return "shape / index argument out of range";
    case BE_ERR_ALIGN: return "pointer not aligned";
    case BE_ERR_UNSUPPORTED: return "request not supported by this build";
    case BE_ERR_NOMEM: return "scratch allocation failed";
    case BE_ERR_STATIC_LIMIT: return "request exceeds the fixed static scratch of this entry point (see BE_STATIC_EIGH_MAX_ELEMS)";
    default: break;
  }
  if (code > 0) return cudaGetErrorString((cudaError_t)code);
  return "unknown error";
}

extern "C" int be_set_workspace_limit(be_ctx* ctx, size_t bytes) {
  BE_DEVICE_GUARD(ctx);
  if (!ctx) return BE_ERR_NULL;
  if (bytes < ((size_t)1 << 20)) return BE_ERR_SHAPE;
  ctx->ws_limit = bytes;
  ctx->ws_user = 1;
  return BE_OK;
}

extern "C" int be_set_chunk_pipeline(be_ctx* ctx, int on) {
  BE_DEVICE_GUARD(ctx);
  if (!ctx) return BE_ERR_NULL;
  ctx->chunk_pipeline = on ? 1 : 0;
  return BE_OK;
}

extern "C" int be_set_eigh_algorithm(be_ctx* ctx, int algo) {
  BE_DEVICE_GUARD(ctx);
  if (!ctx) return BE_ERR_NULL;
  if (algo < 0 || algo > 2) return BE_ERR_SHAPE;
  ctx->eigh_algo = algo;
  return BE_OK;
}

extern "C" int be_release_workspace(be_ctx* ctx) {
  BE_DEVICE_GUARD(ctx);
  if (!ctx) return BE_ERR_NULL;
  BE_CUDA(cudaStreamSynchronize(ctx->stream));
  if (ctx->copy_stream) BE_CUDA(cudaStreamSynchronize(ctx->copy_stream));
  if (ctx->arena) { cudaFree(ctx->arena); ctx->arena = nullptr; ctx->arena_bytes = 0; ctx->arena_used = 0; }
  for (int i = 0; i < 2; ++i) if (ctx->stage_buf[i]) { cudaFree(ctx->stage_buf[i]); ctx->stage_buf[i] = nullptr; }
  ctx->stage_cap[0] = ctx->stage_cap[1] = 0;
  return BE_OK;
}

extern "C" int64_t be_launch_count(const be_ctx* ctx) {
  BE_DEVICE_GUARD(ctx); return ctx ? ctx->launches : 0; }

extern "C" int64_t be_host_grid_bytes_copied(const be_ctx* ctx) { return ctx ? ctx->h2d_bytes : 0; }
extern "C" int be_host_schedule(const be_ctx* ctx) { return ctx ? ctx->host_schedule : 0; }

// ---------------------------------------------------------------------------------------------
size_t be_eigh_scratch_bytes(int64_t cnt, int N, int nv) {
  if (N <= 8) return 256 + (size_t)cnt * N * N * sizeof(cplx);   // (+ the assembled chunk of a *_bloch call)
  if (N <= TS_MAXN) return be_eigh_large_scratch_bytes(cnt, N, nv) + (size_t)cnt * N * N * sizeof(cplx) + 4096;
  return be_eigh_large_scratch_bytes(cnt, N, nv) + 4096;
}

int be_eigh_frames(be_ctx* ctx, const cplx* H, const GridMap& map, int64_t loop0, int64_t cnt,
                   int N, int nv, int ne, double* E, cplx* X, int* info) {
  if (cnt <= 0) return BE_OK;
  const size_t mark = ctx->arena_used;
  if (ctx->bloch && N <= TS_MAXN) {
    // small matrices: assemble the chunk into a scratch grid, then solve it as a flat batch (the large
    // path assembles straight into its work copy inside be_eigh_large)
    const BlochSrc* bs = ctx->bloch;
    cplx* T = (cplx*)be_arena_alloc(ctx, (size_t)cnt * N * N * sizeof(cplx));
    if (!T) return BE_ERR_NOMEM;
    BE_TRY(be_bloch_assemble_chunk(ctx, bs, loop0, cnt, N, T));
    ctx->bloch = nullptr;
    GridMap fm;
    memset(&fm, 0, sizeof(fm));
    fm.ndim = 1; fm.dir = 0; fm.n1 = 1; fm.dims[0] = 1; fm.batch_stride = 1; fm.loops = cnt;
    const int r = (N <= 8) ? be_eigh_small(ctx, T, fm, 0, cnt, N, nv, E, X, info)
                           : be_eigh_large(ctx, T, fm, 0, cnt, N, nv, ne, E, X, info);
    ctx->bloch = bs;
    ctx->arena_used = mark;
    return r;
  }
  if (N <= 8) return be_eigh_small(ctx, H, map, loop0, cnt, N, nv, E, X, info);
  const int r = be_eigh_large(ctx, H, map, loop0, cnt, N, nv, ne, E, X, info);
  ctx->arena_used = mark;   // stage scratch is dead once its kernels are enqueued (stream order)
  return r;
}

static inline bool aligned(const void* p, size_t a) { return ((uintptr_t)p % a) == 0; }

static GridMap flat_map(int64_t count) {
  GridMap m;
  memset(&m, 0, sizeof(m));
  m.ndim = 1; m.dir = 0; m.n1 = 1; m.shift = 0;
  m.dims[0] = 1; m.stride[0] = 0; m.batch_stride = 1; m.loops = count;
  return m;
}

extern "C" size_t be_workspace_bytes(const be_grid* g, int n_occ, int op) {
  if (!g || g->ndim < 1 || g->ndim > 3) return 0;
  int64_t pts = g->batch;
  for (int a = 0; a < g->ndim; ++a) pts *= g->dims[a];
  const int N = g->N, m = (op == 0) ? n_occ : n_occ;
  size_t per = be_eigh_scratch_bytes(1, N, m) + (size_t)N * (m + 1) * 16 * 4 + (size_t)m * m * 16 * 6;
  size_t tot = per * (size_t)pts;
  const size_t cap = (size_t)64 << 30;
  return tot < cap ? tot : cap;
}

// ---------------------------------------------------------------------------------------------
extern "C" int be_eigh_batched(be_ctx* ctx, const void* dH, int64_t count, int N, int n_vec,
                               double* dE, void* dU, int* d_info) {
  BE_DEVICE_GUARD(ctx);
  if (!ctx) return BE_ERR_NULL;
  if (count < 0 || N < 1 || n_vec < 0 || n_vec > N) return BE_ERR_SHAPE;
  if (count == 0) return BE_OK;
  if (!dH || !dE) return BE_ERR_NULL;
  if (!aligned(dH, 16) || !aligned(dE, 8) || (dU && !aligned(dU, 16))) return BE_ERR_ALIGN;
  if (count == 0) return BE_OK;
  const int nv = dU ? n_vec : 0;
  const size_t per = be_eigh_scratch_bytes(1, N, nv) + (size_t)N * (nv > 0 ? nv : 1) * sizeof(cplx) + 1024;
  int64_t chunk = (int64_t)(be_effective_ws_limit(ctx, per * (size_t)count) / per);
  if (chunk < 1) chunk = 1;
  if (chunk > count) chunk = count;
  const int64_t nchunks = (count + chunk - 1) / chunk;
  chunk = (count + nchunks - 1) / nchunks;
  BE_TRY(be_arena_reserve(ctx, per * (size_t)chunk + (1 << 20)));
  const GridMap map = flat_map(count);
  for (int64_t c0 = 0; c0 < count; c0 += chunk) {
    const int64_t cnt = (count - c0 < chunk) ? count - c0 : chunk;
    ctx->arena_used = 0;
    cplx* X = nullptr;
    if (nv > 0) {
      X = (cplx*)be_arena_alloc(ctx, (size_t)cnt * N * nv * sizeof(cplx));
      if (!X) return BE_ERR_NOMEM;
    }
    BE_TRY(be_eigh_frames(ctx, (const cplx*)dH, map, c0, cnt, N, nv, N, dE + c0 * N, X,
                          d_info ? d_info + c0 : nullptr));
    if (nv > 0) BE_TRY(be_frames_to_public(ctx, X, (cplx*)dU + c0 * (int64_t)N * nv, cnt, N, nv));
  }
  return BE_OK;
}

extern "C" int be_winding(be_ctx* ctx, const double* d_theta, int64_t n_cycles, int n_points, int m,
                          double* d_wind) {
  BE_DEVICE_GUARD(ctx);
  if (!ctx || !d_theta || !d_wind) return BE_ERR_NULL;
  if (n_cycles < 0 || n_points < 1 || m < 1) return BE_ERR_SHAPE;
  if (n_cycles == 0) return BE_OK;
  return be_winding_impl(ctx, d_theta, n_cycles, n_points, m, d_wind);
}

extern "C" int be_zgemm_batched(be_ctx* ctx, int opA, int opB, int M, int N, int K,
                                const double* alpha, const void* dA, int lda, int64_t strideA,
                                const void* dB, int ldb, int64_t strideB,
                                const double* beta, void* dC, int ldc, int64_t strideC, int64_t batch, int lower) {
  BE_DEVICE_GUARD(ctx);
  if (!ctx || !dA || !dB || !dC || !alpha || !beta) return BE_ERR_NULL;
  if (M < 0 || N < 0 || K < 0 || batch < 0 || lda < 1 || ldb < 1 || ldc < 1) return BE_ERR_SHAPE;
  if (!aligned(dA, 16) || !aligned(dB, 16) || !aligned(dC, 16)) return BE_ERR_ALIGN;
  ZgemmParams p = zgemm_simple(M, N, K, (const cplx*)dA, lda, strideA, (const cplx*)dB, ldb, strideB,
                               (cplx*)dC, ldc, strideC, batch);
  p.alpha = mkc(alpha[0], alpha[1]); p.beta = mkc(beta[0], beta[1]); p.lower = lower ? 1 : 0;
  return be_zgemm(ctx, opA, opB, p);
}

// ---------------------------------------------------------------------------------------------
// NEXT-1: H(k) assembly as a GEMM
namespace {
__global__ void k_bloch_coef(const double* __restrict__ t, const int* __restrict__ R, int nd, int nR, int64_t count,
                             cplx* __restrict__ coef) {
  const int64_t idx = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (idx >= count * nR) return;
  const int64_t k = idx / nR;
  const int r = (int)(idx % nR);
  double x = 0.0;
  for (int a = 0; a < nd; ++a) x += t[k * nd + a] * (double)R[r * nd + a];
  double s, c;
  sincospi(2.0 * x, &s, &c);
  coef[idx] = mkc(c, s);
}
}  // namespace

extern "C" int be_bloch_coefficients(be_ctx* ctx, const double* d_t, const int* h_R, int nd, int nR, int64_t count,
                                     void* d_coef) {
  BE_DEVICE_GUARD(ctx);
  if (!ctx || !d_t || !h_R || !d_coef) return BE_ERR_NULL;
  if (nd < 1 || nd > 3 || nR < 1 || count < 0) return BE_ERR_SHAPE;
  if (!aligned(d_t, 8) || !aligned(d_coef, 16)) return BE_ERR_ALIGN;
  if (count == 0) return BE_OK;
  BE_TRY(be_arena_reserve(ctx, (size_t)nR * nd * sizeof(int) + 4096));
  int* dR = (int*)be_arena_alloc(ctx, (size_t)nR * nd * sizeof(int));
  if (!dR) return BE_ERR_NOMEM;
  // small pageable copy: staged by the runtime before the call returns
  BE_CUDA(cudaMemcpyAsync(dR, h_R, (size_t)nR * nd * sizeof(int), cudaMemcpyHostToDevice, ctx->stream));
  const int64_t tot = count * nR;
  k_bloch_coef<<<(unsigned)((tot + 255) / 256), 256, 0, ctx->stream>>>(d_t, dR, nd, nR, count, (cplx*)d_coef);
  ctx->launches++;
  return (int)cudaGetLastError();
}

extern "C" int be_assemble_bloch(be_ctx* ctx, const void* dA, const void* d_coef, int64_t count, int N, int nR,
                                 void* dH) {
  BE_DEVICE_GUARD(ctx);
  if (!ctx || !dA || !d_coef || !dH) return BE_ERR_NULL;
  if (N < 1 || nR < 1 || count < 0 || (int64_t)N * N > 0x7fffffffLL || count > 0x7fffffffLL) return BE_ERR_SHAPE;
  if (!aligned(dA, 16) || !aligned(d_coef, 16) || !aligned(dH, 16)) return BE_ERR_ALIGN;
  if (count == 0) return BE_OK;
  // column-major views: A' = dA as (N^2 x nR), B = d_coef as (nR x count), C = dH as (N^2 x count)
  const int M = N * N;
  ZgemmParams g = zgemm_simple(M, (int)count, nR, (const cplx*)dA, M, 0, (const cplx*)d_coef, nR, 0,
                               (cplx*)dH, M, 0, 1);
  return be_zgemm(ctx, BE_OP_N, BE_OP_N, g);
}

// ---------------------------------------------------------------------------------------------
// chunk-wise H(k) generation for the *_bloch entry points
namespace {
__global__ void k_bloch_coef_chunk(const int* __restrict__ R, int nR, GridMap map, int64_t loop0, int64_t cnt,
                                   cplx* __restrict__ coef) {
  const int64_t idx = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (idx >= cnt * nR) return;
  const int64_t c = idx / nR;
  const int r = (int)(idx % nR);
  int64_t rest = loop0 + c / map.n1;
  int j = (int)(c % map.n1) + map.shift;
  if (j >= map.n1) j -= map.n1;
  double x = (double)j / map.n1 * (double)R[r * map.ndim + map.dir];
  for (int a = map.ndim - 1; a >= 0; --a) {
    if (a == map.dir) continue;
    const int64_t i = rest % map.dims[a];
    rest /= map.dims[a];
    x += (double)i / map.dims[a] * (double)R[r * map.ndim + a];
  }
  double s, co;
  sincospi(2.0 * x, &s, &co);
  coef[idx] = mkc(co, s);
}
}  // namespace

int be_bloch_assemble_chunk(be_ctx* ctx, const BlochSrc* bs, int64_t loop0, int64_t cnt, int N, cplx* out) {
  const size_t mark = ctx->arena_used;
  cplx* coef = (cplx*)be_arena_alloc(ctx, (size_t)cnt * bs->nR * sizeof(cplx));
  if (!coef) return BE_ERR_NOMEM;
  const int64_t tot = cnt * bs->nR;
  k_bloch_coef_chunk<<<(unsigned)((tot + 255) / 256), 256, 0, ctx->stream>>>(bs->dR, bs->nR, bs->map, loop0, cnt, coef);
  ctx->launches++;
  BE_CUDA(cudaGetLastError());
  // one GEMM per realization present in the chunk (loops are enumerated batch-major)
  const int n1 = bs->map.n1;
  const int M = N * N;
  int64_t c0 = 0;
  while (c0 < cnt) {
    const int64_t loop = loop0 + c0 / n1;
    const int64_t bt = loop / bs->loops_per_batch;
    int64_t c1 = ((bt + 1) * bs->loops_per_batch - loop0) * n1;   // first matrix of the next realization
    if (c1 > cnt) c1 = cnt;
    ZgemmParams g = zgemm_simple(M, (int)(c1 - c0), bs->nR, bs->A + bt * (int64_t)bs->nR * M, M, 0,
                                 coef + c0 * bs->nR, bs->nR, 0, out + c0 * (int64_t)M, M, 0, 1);
    BE_TRY(be_zgemm(ctx, BE_OP_N, BE_OP_N, g));
    c0 = c1;
  }
  ctx->arena_used = mark;   // coef is dead once the GEMMs are enqueued
  return BE_OK;
}
