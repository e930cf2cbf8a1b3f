#include "tvbx_kernels.h"
namespace tvbx {
KernelPick<float> pick_kernel_f32(bool single, bool closed, int spc) {
  constexpr int MT = MaxT<float>::v;
  if (!closed) return single ? KernelPick<float>{integrate_kernel<float, true, false, 0, MT>} : KernelPick<float>{integrate_kernel<float, false, false, 0, MT>};
#define TVBX_CASE(S) case S: return single ? KernelPick<float>{integrate_kernel<float, true, true, S, MT>} : KernelPick<float>{integrate_kernel<float, false, true, S, MT>};
  switch (spc) {
    TVBX_CASE(1) TVBX_CASE(2) TVBX_CASE(4) TVBX_CASE(7)
    default: break;
  }
#undef TVBX_CASE
  return single ? KernelPick<float>{integrate_kernel<float, true, true, 0, MT>} : KernelPick<float>{integrate_kernel<float, false, true, 0, MT>};
}
}  // namespace tvbx
