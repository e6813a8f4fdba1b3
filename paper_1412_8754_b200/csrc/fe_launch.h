// fe_launch.h -- internal: host-side launchers of the k-sum kernels, one translation unit per tile / block shape so
// that build.py can compile them in parallel (fe_launch_tile.cu, fe_launch_coop.cu); called from fe_api.cu only.
#pragma once
#include <cuda_runtime.h>

#include "fe_ksum_coop.cuh"

namespace fe {

// Per-temperature constants of the extended-range exponential (fe_kernels.cuh), in long double on the host.
inline FactoredConsts make_factored(double T) {
  FactoredConsts fc;
  const long double ln2 = 0.693147180559945309417232121458176568L;
  const long double c2 = (long double)T * ln2 / 256.0L;
  fc.c1 = (double)(256.0L / ((long double)T * ln2));
  fc.c2hi = (double)c2;
  fc.c2lo = (double)(c2 - (long double)fc.c2hi);
  const long double beta = 1.0L / (long double)T;
  fc.b1 = (double)beta;
  fc.b2 = (double)(beta * beta / 2.0L);
  fc.b3 = (double)(beta * beta * beta / 6.0L);
  fc.b4 = (double)(beta * beta * beta * beta / 24.0L);
  return fc;
}

// K1 / K1f, tile index = position in kTiles of fe_api.cu: (8,4) (4,4) (2,8) (1,8) (16,2) (16,4)
#define FE_DECL_TILE(i) \
  cudaError_t launch_ksum_tile_##i(int nb, int form, int mode, int grid, cudaStream_t st, const KsumParams& P);
FE_DECL_TILE(0) FE_DECL_TILE(1) FE_DECL_TILE(2) FE_DECL_TILE(3) FE_DECL_TILE(4) FE_DECL_TILE(5)
#undef FE_DECL_TILE

// K1c, shape index = position in kCoopShapes of fe_api.cu
#define FE_DECL_COOP(i) cudaError_t launch_coop_shape_##i(int nb, int form, int grid, cudaStream_t st, const CoopParams& P); \
  cudaError_t occupancy_coop_shape_##i(int nb, int form, int sym, int* blocks);
FE_DECL_COOP(0) FE_DECL_COOP(1) FE_DECL_COOP(2) FE_DECL_COOP(3) FE_DECL_COOP(4) FE_DECL_COOP(5)
#undef FE_DECL_COOP

}  // namespace fe
