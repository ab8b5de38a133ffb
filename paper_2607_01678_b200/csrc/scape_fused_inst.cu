// scape_fused_inst.cu — instantiations of the streaming kernels (scape_kernels.cuh).
//
// Compiled several times by paper_2607_01678_b200/build.py, once per gradient element type and
// range of R, so that the translation units build in parallel:
//   -DSCAPE_INST_BF16=0|1  -DSCAPE_INST_RLO=a  -DSCAPE_INST_RHI=b  -DSCAPE_INST_TAG=f32_lo|...
// Each unit exports two lookup functions that hand the kernel's address to scape.cu, which
// launches through cudaLaunchKernel: no method arithmetic and no launch logic lives here.
#include "scape_kernels.cuh"

#ifndef SCAPE_INST_TAG
#error "compile with -DSCAPE_INST_TAG=<tag> -DSCAPE_INST_BF16=<0|1> -DSCAPE_INST_RLO=<a> -DSCAPE_INST_RHI=<b>"
#endif

#define SCAPE_CAT2(a, b) a##b
#define SCAPE_CAT(a, b) SCAPE_CAT2(a, b)

namespace scapek {

#if SCAPE_INST_BF16
using InstG = __nv_bfloat16;
#else
using InstG = float;
#endif

namespace {

template <int R>
const void* step_ptr(bool dense, bool msparse, bool clipt) {
  if (dense) return clipt ? (const void*)scape_fused_step_kernel<InstG, R, true, false, true>
                          : (const void*)scape_fused_step_kernel<InstG, R, true, false, false>;
  if (msparse) return clipt ? (const void*)scape_fused_step_kernel<InstG, R, false, true, true>
                            : (const void*)scape_fused_step_kernel<InstG, R, false, true, false>;
  return clipt ? (const void*)scape_fused_step_kernel<InstG, R, false, false, true>
               : (const void*)scape_fused_step_kernel<InstG, R, false, false, false>;
}

template <int R>
const void* tma_ptr(bool clipt, bool rkview, uint32_t* tile_bytes) {
  if constexpr (tma_can_launch<InstG, R>()) {
    *tile_bytes = tma_tile_bytes<InstG, R>();
    // rkview: the grouped form with the rk tables (per-layer refresh); else the flat form with pre + trank
    if (rkview) return clipt ? (const void*)scape_fused_tmag_kernel<InstG, R, true, true> : (const void*)scape_fused_tmag_kernel<InstG, R, false, true>;
    return clipt ? (const void*)scape_fused_tma_kernel<InstG, R, true, false> : (const void*)scape_fused_tma_kernel<InstG, R, false, false>;
  } else {
    *tile_bytes = 0;
    return nullptr;
  }
}

template <int R>
const void* step_dispatch(int r, bool dense, bool msparse, bool clipt) {
  if constexpr (R > SCAPE_INST_RHI) return nullptr;
  else return r == R ? step_ptr<R>(dense, msparse, clipt) : step_dispatch<R + 1>(r, dense, msparse, clipt);
}

template <int R>
const void* tma_dispatch(int r, bool clipt, bool rkview, uint32_t* tile_bytes) {
  if constexpr (R > SCAPE_INST_RHI) { *tile_bytes = 0; return nullptr; }
  else return r == R ? tma_ptr<R>(clipt, rkview, tile_bytes) : tma_dispatch<R + 1>(r, clipt, rkview, tile_bytes);
}

}  // namespace

// register-staged kernel <InstG, R, dense, msparse, clipt>; nullptr when R is outside this unit's range
const void* SCAPE_CAT(fused_step_kernel_, SCAPE_INST_TAG)(int R, bool dense, bool msparse, bool clipt) {
  return step_dispatch<SCAPE_INST_RLO>(R, dense, msparse, clipt);
}

// bulk-copy staged kernel <InstG, R, clipt, rkview> and the bytes of one of its stages; nullptr when the
// instantiation does not exist (R outside the range, or a tile that can never be resident twice per SM)
const void* SCAPE_CAT(fused_tma_kernel_, SCAPE_INST_TAG)(int R, bool clipt, bool rkview, uint32_t* tile_bytes) {
  return tma_dispatch<SCAPE_INST_RLO>(R, clipt, rkview, tile_bytes);
}

}  // namespace scapek
