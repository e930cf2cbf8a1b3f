#include "tvbx_k_inst.h"
namespace tvbx {
Kernel2Fn k2_g4(int spc, bool sring) {
  if (sring) { TVBX_SPC_SWITCH(spc, true, 4, false, false, true, K2_MAXT, false) }
  TVBX_SPC_SWITCH(spc, true, 4, false, false, false, K2_MAXT, false)
}
}  // namespace tvbx
