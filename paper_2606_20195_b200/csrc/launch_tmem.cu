// launch_tmem.cu -- instantiations of the tensor-memory-privatised scatter.  Compiled once per zeta
// (-DSK_TMEM_ZETA=1|2|4|8) so the four families build in parallel; the zeta = 4 unit also holds the
// shape logic and the dispatcher.
#include "kernel_tmem.cuh"
#include "launch.h"

#ifndef SK_TMEM_ZETA
#error "compile with -DSK_TMEM_ZETA=<1|2|4|8>"
#endif

namespace sk {
namespace {

template <int X, int S>
cudaError_t go(const TmemArgs& g, int grid, cudaStream_t st) {
  constexpr int Z = SK_TMEM_ZETA, NW = 4, N = 64 * X * S;
  auto k = k_tmem<Z, X, S, NW>;
  const size_t smem = tmem_smem_bytes(Z, N);
  cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  k<<<grid, (NW + 1) * 32, smem, st>>>(g);
  return cudaGetLastError();
}

cudaError_t dispatch(const TmemArgs& g, int X, int S, int grid, cudaStream_t st) {
  switch (X * 10 + S) {
    case 11: return go<1, 1>(g, grid, st);
    case 12: return go<1, 2>(g, grid, st);
    case 14: return go<1, 4>(g, grid, st);
    case 21: return go<2, 1>(g, grid, st);
    case 22: return go<2, 2>(g, grid, st);
    case 24: return go<2, 4>(g, grid, st);
    case 41: return go<4, 1>(g, grid, st);
    case 42: return go<4, 2>(g, grid, st);
    case 44: return go<4, 4>(g, grid, st);
  }
  return cudaErrorInvalidValue;
}

}  // namespace

#if SK_TMEM_ZETA == 1
cudaError_t launch_tmem_z1(const TmemArgs& g, int X, int S, int grid, cudaStream_t st) { return dispatch(g, X, S, grid, st); }
#elif SK_TMEM_ZETA == 2
cudaError_t launch_tmem_z2(const TmemArgs& g, int X, int S, int grid, cudaStream_t st) { return dispatch(g, X, S, grid, st); }
#elif SK_TMEM_ZETA == 8
cudaError_t launch_tmem_z8(const TmemArgs& g, int X, int S, int grid, cudaStream_t st) { return dispatch(g, X, S, grid, st); }
#elif SK_TMEM_ZETA == 4
cudaError_t launch_tmem_z4(const TmemArgs& g, int X, int S, int grid, cudaStream_t st) { return dispatch(g, X, S, grid, st); }

// widest X (fewest instructions per byte) whose d * X columns fit one lane quadrant; S = n / (64 X) in {1, 2, 4}
bool tmem_shape(int n, int d, int* X, int* S) {
  if (n <= 0 || d <= 0 || n % 64 != 0) return false;
  for (int x = 4; x >= 1; x >>= 1) {
    if ((int64_t)d * x > kTmemCols || (d * x) % 8 != 0 || n % (64 * x) != 0) continue;
    const int s = n / (64 * x);
    if (s != 1 && s != 2 && s != 4) continue;
    *X = x;
    *S = s;
    return true;
  }
  return false;
}

size_t tmem_smem_bytes_for(int zeta, int n) { return tmem_smem_bytes(zeta, n); }
int tmem_rows_per_stage(int n) { return tmem_stage_rows(n); }

cudaError_t launch_tmem_f16(const TmemArgs& g, int zeta, int grid, cudaStream_t st) {
  int X = 0, S = 0;
  if (!tmem_shape(g.s.n, g.d, &X, &S)) return cudaErrorInvalidValue;
  switch (zeta) {
    case 1: return launch_tmem_z1(g, X, S, grid, st);
    case 2: return launch_tmem_z2(g, X, S, grid, st);
    case 4: return launch_tmem_z4(g, X, S, grid, st);
    case 8: return launch_tmem_z8(g, X, S, grid, st);
  }
  return cudaErrorInvalidValue;
}
#endif

}  // namespace sk
