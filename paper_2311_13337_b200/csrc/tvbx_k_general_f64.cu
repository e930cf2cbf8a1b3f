#include "tvbx_kernels.h"
namespace tvbx {
KernelPick<double> pick_kernel_f64(bool single, bool closed) {
  constexpr int MT = MaxT<double>::v;
  if (single) return closed ? KernelPick<double>{integrate_kernel<double, true, true, 0, MT>} : KernelPick<double>{integrate_kernel<double, true, false, 0, MT>};
  return closed ? KernelPick<double>{integrate_kernel<double, false, true, 0, MT>} : KernelPick<double>{integrate_kernel<double, false, false, 0, MT>};
}
}  // namespace tvbx
