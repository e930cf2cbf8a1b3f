#include "tvbx_k_inst.h"
namespace tvbx {
Kernel2Fn k2_g1(int spc) { TVBX_SPC_SWITCH(spc, true, 1, false, false, true, K2_MAXT, false) }
}  // namespace tvbx
