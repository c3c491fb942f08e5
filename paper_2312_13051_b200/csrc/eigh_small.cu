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
