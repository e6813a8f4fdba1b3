// fe_launch_tile.cu -- K1 (direct / windowed) and K1f (factored) instantiations of ONE register tile.
// Compiled once per tile by build.py with -DFE_TILE_ID=i -DFE_TILE_TH=.. -DFE_TILE_TD=..
#include "../../include/fe.h"
#include "../../include/fe_debug.h"
#include "fe_launch.h"

namespace fe {
namespace {

template <int NB, int FORM, int TH, int TD>
cudaError_t launch_ksum_mode(int mode, int grid, cudaStream_t st, const KsumParams& P) {
  if (mode == FE_EVAL_WINDOWED)    fe_ksum_kernel<NB, FORM, TH, TD, 1><<<grid, kThreads, 0, st>>>(P);
  else if (mode == FE_EVAL_DIRECT) fe_ksum_kernel<NB, FORM, TH, TD, 0><<<grid, kThreads, 0, st>>>(P);
  else                             fe_ksum_factored_kernel<NB, FORM, TH, TD><<<grid, kFThreads, 0, st>>>(P, make_factored(P.T));
  return cudaGetLastError();
}

}  // namespace

#define FE_CAT2(a, b) a##b
#define FE_CAT(a, b) FE_CAT2(a, b)
cudaError_t FE_CAT(launch_ksum_tile_, FE_TILE_ID)(int nb, int form, int mode, int grid, cudaStream_t st, const KsumParams& P) {
  constexpr int TH = FE_TILE_TH, TD = FE_TILE_TD;
  if (nb == 1) return form == 0 ? launch_ksum_mode<1, 0, TH, TD>(mode, grid, st, P)
                                : launch_ksum_mode<1, 1, TH, TD>(mode, grid, st, P);
  if (nb == 2) return form == 0 ? launch_ksum_mode<2, 0, TH, TD>(mode, grid, st, P)
                                : launch_ksum_mode<2, 1, TH, TD>(mode, grid, st, P);
  return cudaErrorInvalidConfiguration;     // three-band model: K1c only
}

}  // namespace fe
