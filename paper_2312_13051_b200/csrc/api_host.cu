// Host-buffer (end-to-end) variants: the grid is streamed host -> device in chunks of whole loops
// on a copy stream, double buffered against the compute stream; results are copied back before
// return.  Semantics are those of the device entry points (include/berryeasy_b200.h).
#include "be_common.cuh"
#include <string.h>

size_t be_wilson_per_loop_bytes(int N, int m, int n1, int spin);

namespace {

struct DevBuf {
  void* p = nullptr;
  ~DevBuf() { if (p) cudaFree(p); }
  int alloc(size_t bytes) { return cudaMalloc(&p, bytes ? bytes : 16) == cudaSuccess ? BE_OK : BE_ERR_NOMEM; }
};

int host_run(be_ctx* ctx, const void* hH, const be_grid* grid, int n_occ, int dir, const void* hS,
             int S_is_diag, int m_lo, bool spin, const void* h_close, double* h_a, double* h_b,
             double* h_c) {
  if (!ctx || !hH || !grid) return BE_ERR_NULL;
  if (grid->ndim < 1 || grid->ndim > 3 || grid->batch < 1 || grid->N < 1) return BE_ERR_SHAPE;
  if (dir != grid->ndim - 1) return BE_ERR_UNSUPPORTED;
  if (n_occ < 1 || n_occ > grid->N) return BE_ERR_SHAPE;
  const int N = grid->N, m = n_occ, n1 = grid->dims[dir];
  int64_t loops = grid->batch;
  for (int a = 0; a < grid->ndim - 1; ++a) loops *= grid->dims[a];
  if (spin) {
    if (!hS) return BE_ERR_NULL;
    if (m_lo < 0) m_lo = m / 2;
    if (m_lo > m) return BE_ERR_SHAPE;
  } else if (!h_a) return BE_ERR_NULL;
  if (!ctx->copy_stream) BE_CUDA(cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking));

  const size_t loop_bytes = (size_t)n1 * N * N * sizeof(cplx);
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
  // The chunking, the scratch arena and the single eigenphase solve at the end are those of the device
  // entry points; the chunks' matrices come through two staging buffers filled on the copy stream.
  HostStage hs;
  memset(&hs, 0, sizeof(hs));
  hs.hH = (const char*)hH;
  hs.loop_bytes = loop_bytes;
  for (int i = 0; i < 2; ++i) {
    BE_CUDA(cudaEventCreateWithFlags(&hs.copied[i], cudaEventDisableTiming));
    BE_CUDA(cudaEventCreateWithFlags(&hs.freed[i], cudaEventDisableTiming));
  }
  int rc = be_wilson_host_device(ctx, &hs, loops, n1, N, m, dclose.p,
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
  for (int i = 0; i < 2; ++i) {
    cudaEventDestroy(hs.copied[i]); cudaEventDestroy(hs.freed[i]);
    if (hs.stage[i]) cudaFree(hs.stage[i]);
  }
  return rc;
}

}  // namespace

extern "C" int be_wilson_loop_host(be_ctx* ctx, const void* hH_grid, const be_grid* grid, int n_occ, int dir,
                                   const void* h_close, double* h_theta, double* h_abs, double* h_mingap) {
  return host_run(ctx, hH_grid, grid, n_occ, dir, nullptr, 0, 0, false, h_close, h_theta, h_abs, h_mingap);
}

extern "C" int be_spin_resolved_wilson_host(be_ctx* ctx, const void* hH_grid, const be_grid* grid, int n_occ,
                                            int dir, const void* hS, int S_is_diag, int m_lo,
                                            const void* h_close, double* h_theta_lo, double* h_theta_hi,
                                            double* h_pso) {
  return host_run(ctx, hH_grid, grid, n_occ, dir, hS, S_is_diag, m_lo, true, h_close, h_theta_lo,
                  h_theta_hi, h_pso);
}
