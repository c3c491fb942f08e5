// S1' -- many-small-matrix regime (N <= 8): cyclic one-sided (Hestenes) Jacobi (jacobi.cuh), one thread per
// matrix, everything in registers / local memory.
#include "jacobi.cuh"

namespace {

template <int N>
__global__ void __launch_bounds__(128) k_jacobi(const cplx* __restrict__ H, GridMap map, int64_t loop0,
                                                int64_t cnt, int nv, double* __restrict__ E,
                                                cplx* __restrict__ X, int* __restrict__ info) {
  const int64_t c = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (c >= cnt) return;
  const int64_t src = gridmap_index(map, loop0 + c / map.n1, (int)(c % map.n1));
  const cplx* h = H + src * (N * N);
  cplx V[N][N];   // [column][row]
  double ev[N];
  int ord[N];
  const bool done = jacobi_hermitian<N>(h, ev, V, ord);
  if (info) info[c] = done ? 0 : 1;
#pragma unroll
  for (int j = 0; j < N; ++j) {
    double val = 0.0;
#pragma unroll
    for (int a = 0; a < N; ++a) if (ord[j] == a) val = ev[a];
    E[c * N + j] = val;
  }
  if (X) {
#pragma unroll
    for (int j = 0; j < N; ++j) {
      if (j < nv) {
#pragma unroll
        for (int a = 0; a < N; ++a)
          if (ord[j] == a) {
            // normalise (V is unitary up to rounding; re-normalise the column)
            double nn = 0.0;
#pragma unroll
            for (int r = 0; r < N; ++r) nn += cabs2(V[a][r]);
            const double sc = 1.0 / sqrt(nn);
#pragma unroll
            for (int r = 0; r < N; ++r) X[c * (int64_t)(N * nv) + j * N + r] = cscale(sc, V[a][r]);
          }
      }
    }
  }
}

}  // namespace

int be_eigh_small(be_ctx* ctx, const cplx* H, const GridMap& map, int64_t loop0, int64_t cnt, int N,
                  int nv, double* E, cplx* X, int* info) {
  const unsigned blocks = (unsigned)((cnt + 127) / 128);
  cudaStream_t st = ctx->stream;
  be_prof_begin(ctx, PK_JACOBI);
  switch (N) {
#define CASE(n) case n: k_jacobi<n><<<blocks, 128, 0, st>>>(H, map, loop0, cnt, nv, E, X, info); break;
    CASE(1) CASE(2) CASE(3) CASE(4) CASE(5) CASE(6) CASE(7) CASE(8)
#undef CASE
    default: return BE_ERR_UNSUPPORTED;
  }
  be_prof_end(ctx, PK_JACOBI, (double)cnt * N * (N + (double)nv + 1) * 16.0, 0.0);
  ctx->launches++;
  return (int)cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------
// be_eigh_batched_static: the N <= 8 eigensolver for callers that must not allocate (CUDA graph capture, serving
// loops, harnesses that forbid cudaMalloc).  k_jacobi writes its frames X [count][n_vec][N] to scratch before they
// are transposed to the public layout; here that scratch is a file-scope device array, resident on every GPU that
// loads the library until the process exits, instead of the context arena.  In host code the array's name is a
// host-side shadow symbol, not a device address: the address is taken with cudaGetSymbolAddress, once per device,
// with that device current.
#include <mutex>
#include <string.h>

static __device__ __align__(256) unsigned char g_static_frames[BE_STATIC_EIGH_MAX_ELEMS * sizeof(cplx)];

namespace {
constexpr int STATIC_MAX_DEVICES = 64;
std::mutex g_static_mu;
void* g_static_ptr[STATIC_MAX_DEVICES] = {nullptr};

// device address of g_static_frames on the CURRENT device (the caller holds the device guard)
int static_frames_ptr(int device, cplx** out) {
  if (device < 0 || device >= STATIC_MAX_DEVICES) return BE_ERR_UNSUPPORTED;
  std::lock_guard<std::mutex> lk(g_static_mu);
  if (!g_static_ptr[device]) {
    void* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&p, g_static_frames);
    if (e != cudaSuccess) return (int)e;
    if (!p) return BE_ERR_NOMEM;
    g_static_ptr[device] = p;
  }
  *out = (cplx*)g_static_ptr[device];
  return BE_OK;
}
}  // namespace

extern "C" int be_eigh_batched_static(be_ctx* ctx, const void* dH, int64_t count, int N, int n_vec, double* dE,
                                      void* dU, int* d_info) {
  BE_DEVICE_GUARD(ctx);
  if (!ctx) return BE_ERR_NULL;
  if (count < 0 || N < 1 || n_vec < 0 || n_vec > N) return BE_ERR_SHAPE;
  if (N > 8) return BE_ERR_UNSUPPORTED;
  if (count == 0) return BE_OK;
  if (!dH || !dE) return BE_ERR_NULL;
  if (((uintptr_t)dH % 16) || ((uintptr_t)dE % 8) || (dU && ((uintptr_t)dU % 16))) return BE_ERR_ALIGN;
  const int nv = dU ? n_vec : 0;
  if (count > (int64_t)BE_STATIC_EIGH_MAX_ELEMS || count * (int64_t)N * (nv > 0 ? nv : 1) > (int64_t)BE_STATIC_EIGH_MAX_ELEMS)
    return BE_ERR_STATIC_LIMIT;
  cplx* X = nullptr;
  if (nv > 0) BE_TRY(static_frames_ptr(ctx->device, &X));
  GridMap fm;
  memset(&fm, 0, sizeof(fm));
  fm.ndim = 1; fm.dir = 0; fm.n1 = 1; fm.shift = 0; fm.dims[0] = 1; fm.stride[0] = 0; fm.batch_stride = 1; fm.loops = count;
  // every frame element in [0, count * nv * N) is written by k_jacobi before k_x2u reads it: nothing to clear
  BE_TRY(be_eigh_small(ctx, (const cplx*)dH, fm, 0, count, N, nv, dE, X, d_info));
  if (nv > 0) BE_TRY(be_frames_to_public(ctx, X, (cplx*)dU, count, N, nv));
  return BE_OK;
}
