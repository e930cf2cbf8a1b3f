#include "tvbx_kernels.h"
#include "tvbx_integrate2_ws.cuh"
namespace tvbx {
// grouped low-latency form: the regions of a group of simulations split over several CTAs (cfg 4: 7 simulations over 4 CTAs)
Kernel2Fn k2_wsg(int spc) {
  switch (spc) {
    case 1: return integrate2_ws_kernel<1, false, true>;
    case 2: return integrate2_ws_kernel<2, false, true>;
    case 3: return integrate2_ws_kernel<3, false, true>;
    case 4: return integrate2_ws_kernel<4, false, true>;
    case 5: return integrate2_ws_kernel<5, false, true>;
    case 6: return integrate2_ws_kernel<6, false, true>;
    case 7: return integrate2_ws_kernel<7, false, true>;
    default: return integrate2_ws_kernel<8, false, true>;
  }
}
}  // namespace tvbx
