#include "tvbx_k_inst.h"
namespace tvbx {
Kernel2Fn k2_g8_small(int spc, bool isamp) {
  if (isamp) { TVBX_SPC_SWITCH(spc, true, 8, false, false, false, K2_SMALLT, true) }
  TVBX_SPC_SWITCH(spc, true, 8, false, false, false, K2_SMALLT, false)
}
// the group's history ring in shared memory for the whole launch (small sweeps whose ring fits: cfg 1)
Kernel2Fn k2_g8_small_sring(int spc) { TVBX_SPC_SWITCH(spc, true, 8, false, false, true, K2_SMALLT, false) }
}  // namespace tvbx
