#include "tvbx_k_inst.h"
namespace tvbx {
Kernel2Fn k2_g8_small(int spc, bool isamp) {
  if (isamp) { TVBX_SPC_SWITCH(spc, true, 8, false, false, false, K2_SMALLT, true) }
  TVBX_SPC_SWITCH(spc, true, 8, false, false, false, K2_SMALLT, false)
}
}  // namespace tvbx
