#include "tvbx_kernels.h"
#include "tvbx_integrate2_ws.cuh"
namespace tvbx {
#define TVBX_WS_SWITCH(spc, SR)                                     \
  switch (spc) {                                                    \
    case 1: return integrate2_ws_kernel<1, SR>;                     \
    case 2: return integrate2_ws_kernel<2, SR>;                     \
    case 3: return integrate2_ws_kernel<3, SR>;                     \
    case 4: return integrate2_ws_kernel<4, SR>;                     \
    case 5: return integrate2_ws_kernel<5, SR>;                     \
    case 6: return integrate2_ws_kernel<6, SR>;                     \
    case 7: return integrate2_ws_kernel<7, SR>;                     \
    default: return integrate2_ws_kernel<8, SR>;                    \
  }
Kernel2Fn k2_ws(int spc, bool sring) {
  if (sring) { TVBX_WS_SWITCH(spc, true) }
  TVBX_WS_SWITCH(spc, false)
}
int k2_ws_max_threads() { return K2_WST; }
}  // namespace tvbx
