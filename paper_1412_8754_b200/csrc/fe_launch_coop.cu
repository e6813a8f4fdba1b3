// fe_launch_coop.cu -- K1c instantiations of ONE block shape.  Compiled once per shape by build.py with
// -DFE_COOP_ID=i -DFE_COOP_TH=.. -DFE_COOP_TD=.. -DFE_COOP_LH=.. -DFE_COOP_NW=.. -DFE_COOP_KB=.. -DFE_COOP_MINB=..
#include "../../include/fe.h"
#include "../../include/fe_debug.h"
#include "fe_launch.h"

namespace fe {
namespace {

template <int NB, int FORM, int TH, int TD, int LH, int NW, int KB, int MINB, int SYM>
cudaError_t launch_coop_sym(int grid, cudaStream_t st, const CoopParams& P) {
  using G = CoopGeom<TH, TD, LH, NW, KB, NB>;
  auto kern = fe_ksum_coop_kernel<NB, FORM, TH, TD, LH, NW, KB, MINB, SYM>;
  // The opt-in is per DEVICE (and a handle binds to the device current at fe_create), so it is set before every
  // launch: a host-side call of a few hundred nanoseconds, no static state shared between devices or host threads.
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)G::smem_bytes);
  if (e != cudaSuccess) return e;
  kern<<<grid, G::NT, G::smem_bytes, st>>>(P);
  return cudaGetLastError();
}

template <int NB, int FORM, int TH, int TD, int LH, int NW, int KB, int MINB>
cudaError_t launch_coop_inst(int grid, cudaStream_t st, const CoopParams& P) {
  if constexpr (NB < 3) {           // symmetry-reduced k set (fe_set_symmetry): one- and two-band models
    if (P.sym != 0) return launch_coop_sym<NB, FORM, TH, TD, LH, NW, KB, MINB, 1>(grid, st, P);
  }
  return launch_coop_sym<NB, FORM, TH, TD, LH, NW, KB, MINB, 0>(grid, st, P);
}

template <int TH, int TD, int LH, int NW, int KB, int MINB>
cudaError_t launch_coop_shape(int nb, int form, int grid, cudaStream_t st, const CoopParams& P) {
  if constexpr (LH == 4) {          // three-band model: the LH = 4 shapes only (fused-P1 slot mapping, fe_ksum_coop.cuh)
    if (nb == 3) return form == 0 ? launch_coop_inst<3, 0, TH, TD, LH, NW, KB, MINB>(grid, st, P)
                                  : launch_coop_inst<3, 1, TH, TD, LH, NW, KB, MINB>(grid, st, P);
  }
  if (nb == 3) return cudaErrorInvalidConfiguration;
  if (nb == 1) return form == 0 ? launch_coop_inst<1, 0, TH, TD, LH, NW, KB, MINB>(grid, st, P)
                                : launch_coop_inst<1, 1, TH, TD, LH, NW, KB, MINB>(grid, st, P);
  return form == 0 ? launch_coop_inst<2, 0, TH, TD, LH, NW, KB, MINB>(grid, st, P)
                   : launch_coop_inst<2, 1, TH, TD, LH, NW, KB, MINB>(grid, st, P);
}

}  // namespace

// Resident blocks per SM of one instance on the current device (cudaOccupancyMaxActiveBlocksPerMultiprocessor with the
// instance's dynamic shared memory): lets a test catch an instance that silently stopped fitting its launch bound.
template <int NB, int FORM, int TH, int TD, int LH, int NW, int KB, int MINB, int SYM>
cudaError_t occupancy_coop_sym(int* blocks) {
  using G = CoopGeom<TH, TD, LH, NW, KB, NB>;
  auto kern = fe_ksum_coop_kernel<NB, FORM, TH, TD, LH, NW, KB, MINB, SYM>;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)G::smem_bytes);
  if (e != cudaSuccess) return e;
  return cudaOccupancyMaxActiveBlocksPerMultiprocessor(blocks, kern, G::NT, G::smem_bytes);
}

template <int TH, int TD, int LH, int NW, int KB, int MINB>
cudaError_t occupancy_coop_shape(int nb, int form, int sym, int* blocks) {
#define FE_OCC(NB_, F_) (sym ? occupancy_coop_sym<NB_, F_, TH, TD, LH, NW, KB, MINB, 1>(blocks) \
                             : occupancy_coop_sym<NB_, F_, TH, TD, LH, NW, KB, MINB, 0>(blocks))
  if constexpr (LH == 4) {
    if (nb == 3) return form == 0 ? occupancy_coop_sym<3, 0, TH, TD, LH, NW, KB, MINB, 0>(blocks)
                                  : occupancy_coop_sym<3, 1, TH, TD, LH, NW, KB, MINB, 0>(blocks);
  }
  if (nb == 3) return cudaErrorInvalidConfiguration;
  if (nb == 1) return form == 0 ? FE_OCC(1, 0) : FE_OCC(1, 1);
  return form == 0 ? FE_OCC(2, 0) : FE_OCC(2, 1);
#undef FE_OCC
}

#define FE_CAT2(a, b) a##b
#define FE_CAT(a, b) FE_CAT2(a, b)
cudaError_t FE_CAT(launch_coop_shape_, FE_COOP_ID)(int nb, int form, int grid, cudaStream_t st, const CoopParams& P) {
  return launch_coop_shape<FE_COOP_TH, FE_COOP_TD, FE_COOP_LH, FE_COOP_NW, FE_COOP_KB, FE_COOP_MINB>(nb, form, grid, st, P);
}
cudaError_t FE_CAT(occupancy_coop_shape_, FE_COOP_ID)(int nb, int form, int sym, int* blocks) {
  return occupancy_coop_shape<FE_COOP_TH, FE_COOP_TD, FE_COOP_LH, FE_COOP_NW, FE_COOP_KB, FE_COOP_MINB>(nb, form, sym, blocks);
}

}  // namespace fe
