// Host-buffer (end-to-end) variants: the grid is streamed host -> device in chunks of whole loops
// on a copy stream, double buffered against the compute stream; results are copied back before
// return.  Semantics are those of the device entry points (include/berryeasy_b200.h).
#include "be_common.cuh"
#include <string.h>

namespace {

struct DevBuf {
  void* p = nullptr;
  ~DevBuf() { if (p) cudaFree(p); }
  int alloc(size_t bytes) { return cudaMalloc(&p, bytes ? bytes : 16) == cudaSuccess ? BE_OK : BE_ERR_NOMEM; }
};

// the four events of a HostStage, destroyed on every exit path
struct StageEvents {
  HostStage* hs;
  bool ok = true;
  explicit StageEvents(HostStage* h) : hs(h) {
    for (int i = 0; i < 2; ++i) {
      hs->copied[i] = nullptr; hs->freed[i] = nullptr;
      ok = ok && cudaEventCreateWithFlags(&hs->copied[i], cudaEventDisableTiming) == cudaSuccess;
      ok = ok && cudaEventCreateWithFlags(&hs->freed[i], cudaEventDisableTiming) == cudaSuccess;
    }
  }
  ~StageEvents() {
    for (int i = 0; i < 2; ++i) {
      if (hs->copied[i]) cudaEventDestroy(hs->copied[i]);
      if (hs->freed[i]) cudaEventDestroy(hs->freed[i]);
    }
  }
};

// both streams are drained on every exit path: nothing of this call is in flight when it returns
struct DrainStreams {
  be_ctx* ctx;
  ~DrainStreams() { if (ctx->copy_stream) cudaStreamSynchronize(ctx->copy_stream); cudaStreamSynchronize(ctx->stream); }
};

int host_run(be_ctx* ctx, const void* hH, const be_grid* grid, int n_occ, int dir, const void* hS,
             int S_is_diag, int m_lo, bool spin, const void* h_close, double* h_a, double* h_b,
             double* h_c) {
  if (!ctx || !hH || !grid) return BE_ERR_NULL;
  if (grid->ndim < 1 || grid->ndim > 3 || grid->batch < 1 || grid->N < 1) return BE_ERR_SHAPE;
  if (dir < 0 || dir >= grid->ndim) return BE_ERR_SHAPE;
  if (n_occ < 1 || n_occ > grid->N) return BE_ERR_SHAPE;
  const int N = grid->N, m = n_occ, n1 = grid->dims[dir];
  int64_t loops = grid->batch;
  for (int a = 0; a < grid->ndim; ++a) if (a != dir) loops *= grid->dims[a];
  if (spin) {
    if (!hS) return BE_ERR_NULL;
    if (m_lo < 0) m_lo = m / 2;
    if (m_lo > m) return BE_ERR_SHAPE;
  } else if (!h_a) return BE_ERR_NULL;
  int prev_dev = 0;
  BE_CUDA(cudaGetDevice(&prev_dev));
  BE_CUDA(cudaSetDevice(ctx->device));
  struct Restore { int d; ~Restore() { cudaSetDevice(d); } } restore{prev_dev};
  if (!ctx->copy_stream) BE_CUDA(cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking));
  DrainStreams drain{ctx};

  DevBuf dS, dclose, da, db, dc;
  const int mlo = spin ? m_lo : 0, mhi = spin ? m - m_lo : 0;
  if (spin) {
    const size_t sb = S_is_diag ? (size_t)N * sizeof(double) : (size_t)N * N * sizeof(cplx);
    BE_TRY(dS.alloc(sb));
    BE_CUDA(cudaMemcpyAsync(dS.p, hS, sb, cudaMemcpyHostToDevice, ctx->stream));
    if (h_a) BE_TRY(da.alloc((size_t)loops * mlo * sizeof(double)));
    if (h_b) BE_TRY(db.alloc((size_t)loops * mhi * sizeof(double)));
    if (h_c) BE_TRY(dc.alloc((size_t)loops * n1 * m * sizeof(double)));
  } else {
    BE_TRY(da.alloc((size_t)loops * m * sizeof(double)));
    if (h_b) BE_TRY(db.alloc((size_t)loops * m * sizeof(double)));
    if (h_c) BE_TRY(dc.alloc((size_t)loops * sizeof(double)));
  }
  if (h_close) {
    BE_TRY(dclose.alloc((size_t)N * sizeof(cplx)));
    BE_CUDA(cudaMemcpyAsync(dclose.p, h_close, (size_t)N * sizeof(cplx), cudaMemcpyHostToDevice, ctx->stream));
  }
  // The scratch arena and the single eigenphase solve at the end are those of the device entry points; the
  // chunks' matrices come through two staging buffers filled on the copy stream.
  HostStage hs;
  memset(&hs, 0, sizeof(hs));
  hs.hH = (const char*)hH;
  hs.mat_bytes = (size_t)N * N * sizeof(cplx);
  hs.loop_bytes = (size_t)n1 * hs.mat_bytes;
  StageEvents ev(&hs);
  if (!ev.ok) return (int)cudaGetLastError();
  int rc = be_wilson_host_device(ctx, &hs, grid, dir, m, dclose.p,
                                 spin ? nullptr : (double*)da.p, spin ? nullptr : (double*)db.p,
                                 spin ? nullptr : (double*)dc.p, dS.p, S_is_diag, m_lo,
                                 spin ? (double*)da.p : nullptr, spin ? (double*)db.p : nullptr,
                                 spin ? (double*)dc.p : nullptr, spin ? 1 : 0);
  if (rc == BE_OK) {
    cudaStream_t st = ctx->stream;
    if (spin) {
      if (h_a && rc == BE_OK) rc = (int)cudaMemcpyAsync(h_a, da.p, (size_t)loops * mlo * sizeof(double), cudaMemcpyDeviceToHost, st);
      if (h_b && rc == BE_OK) rc = (int)cudaMemcpyAsync(h_b, db.p, (size_t)loops * mhi * sizeof(double), cudaMemcpyDeviceToHost, st);
      if (h_c && rc == BE_OK) rc = (int)cudaMemcpyAsync(h_c, dc.p, (size_t)loops * n1 * m * sizeof(double), cudaMemcpyDeviceToHost, st);
    } else {
      rc = (int)cudaMemcpyAsync(h_a, da.p, (size_t)loops * m * sizeof(double), cudaMemcpyDeviceToHost, st);
      if (h_b && rc == BE_OK) rc = (int)cudaMemcpyAsync(h_b, db.p, (size_t)loops * m * sizeof(double), cudaMemcpyDeviceToHost, st);
      if (h_c && rc == BE_OK) rc = (int)cudaMemcpyAsync(h_c, dc.p, (size_t)loops * sizeof(double), cudaMemcpyDeviceToHost, st);
    }
  }
  cudaStreamSynchronize(ctx->copy_stream);
  const cudaError_t se = cudaStreamSynchronize(ctx->stream);
  if (rc == BE_OK && se != cudaSuccess) rc = (int)se;
  return rc;
}

}  // namespace

extern "C" int be_wilson_loop_host(be_ctx* ctx, const void* hH_grid, const be_grid* grid, int n_occ, int dir,
                                   const void* h_close, double* h_theta, double* h_abs, double* h_mingap) {
  BE_DEVICE_GUARD(ctx);
  return host_run(ctx, hH_grid, grid, n_occ, dir, nullptr, 0, 0, false, h_close, h_theta, h_abs, h_mingap);
}

extern "C" int be_spin_resolved_wilson_host(be_ctx* ctx, const void* hH_grid, const be_grid* grid, int n_occ,
                                            int dir, const void* hS, int S_is_diag, int m_lo,
                                            const void* h_close, double* h_theta_lo, double* h_theta_hi,
                                            double* h_pso) {
  BE_DEVICE_GUARD(ctx);
  return host_run(ctx, hH_grid, grid, n_occ, dir, hS, S_is_diag, m_lo, true, h_close, h_theta_lo,
                  h_theta_hi, h_pso);
}

// Nested loop on a host grid: both levels need the whole plane, so the grid is copied in one piece (it has to
// fit next to the workspace), the device entry point runs, the phases come back.
extern "C" int be_nested_wilson_host(be_ctx* ctx, const void* hH_grid, const be_grid* grid, int n_occ, int dir1, int dir2,
                                     int base, int wb_lo, int wb_hi, double theta_cut, const void* h_close1,
                                     const void* h_close2, double* h_theta1, double* h_theta_nested) {
  BE_DEVICE_GUARD(ctx);
  if (!ctx || !hH_grid || !grid || !h_theta_nested) return BE_ERR_NULL;
  if (grid->ndim < 2 || grid->ndim > 3 || grid->batch < 1 || grid->N < 1) return BE_ERR_SHAPE;
  if (dir1 < 0 || dir1 >= grid->ndim || dir2 < 0 || dir2 >= grid->ndim || dir1 == dir2) return BE_ERR_SHAPE;
  if (wb_lo < 0 || wb_hi > n_occ || wb_lo >= wb_hi) return BE_ERR_SHAPE;
  int prev_dev = 0;
  BE_CUDA(cudaGetDevice(&prev_dev));
  BE_CUDA(cudaSetDevice(ctx->device));
  struct Restore { int d; ~Restore() { cudaSetDevice(d); } } restore{prev_dev};
  DrainStreams drain{ctx};
  const int N = grid->N;
  int64_t pts = grid->batch, loops = grid->batch, outer2 = grid->batch;
  for (int a = 0; a < grid->ndim; ++a) {
    pts *= grid->dims[a];
    if (a != dir1) loops *= grid->dims[a];
    if (a != dir1 && a != dir2) outer2 *= grid->dims[a];
  }
  const int ns = wb_hi - wb_lo;
  DevBuf dH, dc1, dc2, dth1, dthn;
  BE_TRY(dH.alloc((size_t)pts * N * N * sizeof(cplx)));
  BE_TRY(dthn.alloc((size_t)outer2 * ns * sizeof(double)));
  if (h_theta1) BE_TRY(dth1.alloc((size_t)loops * n_occ * sizeof(double)));
  cudaStream_t st = ctx->stream;
  BE_CUDA(cudaMemcpyAsync(dH.p, hH_grid, (size_t)pts * N * N * sizeof(cplx), cudaMemcpyHostToDevice, st));
  ctx->h2d_bytes += (int64_t)pts * N * N * (int64_t)sizeof(cplx);
  if (h_close1) { BE_TRY(dc1.alloc((size_t)N * sizeof(cplx))); BE_CUDA(cudaMemcpyAsync(dc1.p, h_close1, (size_t)N * sizeof(cplx), cudaMemcpyHostToDevice, st)); }
  if (h_close2) { BE_TRY(dc2.alloc((size_t)N * sizeof(cplx))); BE_CUDA(cudaMemcpyAsync(dc2.p, h_close2, (size_t)N * sizeof(cplx), cudaMemcpyHostToDevice, st)); }
  BE_TRY(be_nested_wilson(ctx, dH.p, grid, n_occ, dir1, dir2, base, wb_lo, wb_hi, theta_cut, dc1.p, dc2.p,
                          (double*)dth1.p, (double*)dthn.p));
  BE_CUDA(cudaMemcpyAsync(h_theta_nested, dthn.p, (size_t)outer2 * ns * sizeof(double), cudaMemcpyDeviceToHost, st));
  if (h_theta1) BE_CUDA(cudaMemcpyAsync(h_theta1, dth1.p, (size_t)loops * n_occ * sizeof(double), cudaMemcpyDeviceToHost, st));
  BE_CUDA(cudaStreamSynchronize(st));
  return BE_OK;
}
