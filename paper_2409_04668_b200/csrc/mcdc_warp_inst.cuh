// mcdc_warp_inst.cuh -- launch table of k_warp.  The 48 instantiations <STAGED, RECORD, VARIANT, SCORE> and the 16 for general
// CSG regions <STAGED, RECORD, VARIANT, 0, RGN = true> are compiled in
// four translation units (mcdc_warp_inst.cu with -DMCDC_WARP_VARIANT=0..3, built in parallel); mcdc_host.cu sees only
// the declarations below.
#pragma once
#include "mcdc_warp.cuh"

#ifndef MCDC_WARP_THREADS
#define MCDC_WARP_THREADS 512               // threads per block of k_warp (a compile-time choice: 16 warps x 128 registers)
#endif

namespace mcdc {

// score < 0: the instantiation for general CSG regions (SCORE = 0, RGN = true)
template <int VARIANT>
void warp_launch_variant(bool staged, bool record, int score, int grid, size_t smem, cudaStream_t st, const Tables &T,
                         const HistoryArgs &A);
template <int VARIANT>
cudaError_t warp_set_smem_variant(bool staged, bool record, int score, int bytes);

#ifdef MCDC_WARP_VARIANT
namespace detail {
template <bool STAGED, bool RECORD, int VARIANT, int SCORE, bool RGN = false>
struct WarpInst {
  static void launch(int grid, size_t smem, cudaStream_t st, const Tables &T, const HistoryArgs &A) {
    k_warp<STAGED, RECORD, VARIANT, SCORE, MCDC_WARP_THREADS, RGN><<<grid, MCDC_WARP_THREADS, smem, st>>>(T, A);
  }
  static cudaError_t set_smem(int bytes) {
    return cudaFuncSetAttribute(k_warp<STAGED, RECORD, VARIANT, SCORE, MCDC_WARP_THREADS, RGN>,
                                cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
  }
};
// F(WarpInst<...>) for the run-time choice (staged, record, score)
template <int VARIANT, class F>
auto warp_dispatch(bool staged, bool record, int score, F f) {
#define MCDC_ROW(ST, RC)                                                     \
  switch (score) {                                                          \
    case -1: return f(WarpInst<ST, RC, VARIANT, 0, true>());                 \
    case 0: return f(WarpInst<ST, RC, VARIANT, 0>());                        \
    case 1: return f(WarpInst<ST, RC, VARIANT, 1>());                        \
    default: return f(WarpInst<ST, RC, VARIANT, 2>());                       \
  }
  if (staged) { if (record) { MCDC_ROW(true, true) } else { MCDC_ROW(true, false) } }
  else        { if (record) { MCDC_ROW(false, true) } else { MCDC_ROW(false, false) } }
#undef MCDC_ROW
}
}  // namespace detail

template <int VARIANT>
void warp_launch_variant(bool staged, bool record, int score, int grid, size_t smem, cudaStream_t st, const Tables &T,
                         const HistoryArgs &A) {
  detail::warp_dispatch<VARIANT>(staged, record, score, [&](auto inst) { decltype(inst)::launch(grid, smem, st, T, A); return 0; });
}
template <int VARIANT>
cudaError_t warp_set_smem_variant(bool staged, bool record, int score, int bytes) {
  return detail::warp_dispatch<VARIANT>(staged, record, score, [&](auto inst) { return decltype(inst)::set_smem(bytes); });
}
template void warp_launch_variant<MCDC_WARP_VARIANT>(bool, bool, int, int, size_t, cudaStream_t, const Tables &, const HistoryArgs &);
template cudaError_t warp_set_smem_variant<MCDC_WARP_VARIANT>(bool, bool, int, int);
#endif

}  // namespace mcdc
