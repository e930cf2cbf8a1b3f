#include "tvbx_k_inst.h"
namespace tvbx {
Kernel2Fn k2_g8(int spc, bool isamp) {
  if (isamp) { TVBX_SPC_SWITCH(spc, true, 8, false, false, false, K2_MAXT, true) }
  TVBX_SPC_SWITCH(spc, true, 8, false, false, false, K2_MAXT, false)
}
}  // namespace tvbx
