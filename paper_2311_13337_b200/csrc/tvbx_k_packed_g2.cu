#include "tvbx_k_inst.h"
namespace tvbx {
Kernel2Fn k2_g2(int spc, bool sring) {
  if (sring) { TVBX_SPC_SWITCH(spc, true, 2, false, false, true, K2_MAXT, false) }
  TVBX_SPC_SWITCH(spc, true, 2, false, false, false, K2_MAXT, false)
}
}  // namespace tvbx
