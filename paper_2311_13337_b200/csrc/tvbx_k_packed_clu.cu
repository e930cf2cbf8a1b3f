#include "tvbx_k_inst.h"
namespace tvbx {
Kernel2Fn k2_clu(int spc) { TVBX_SPC_SWITCH(spc, false, 8, true, false, false, K2_MAXT, false) }
Kernel2Fn k2_clu_small(int spc) { TVBX_SPC_SWITCH(spc, true, 8, true, false, false, K2_SMALLT, false) }
Kernel2Fn k2_vec(int spc, bool smemtab) {
  if (smemtab) return spc == 8 ? integrate2_kernel<8, true, 8, true, true, false, K2_MAXT, false> : integrate2_kernel<4, true, 8, true, true, false, K2_MAXT, false>;
  return spc == 8 ? integrate2_kernel<8, false, 8, true, true, false, K2_MAXT, false> : integrate2_kernel<4, false, 8, true, true, false, K2_MAXT, false>;
}
}  // namespace tvbx
