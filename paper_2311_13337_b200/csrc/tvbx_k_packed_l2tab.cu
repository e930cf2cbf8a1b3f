#include "tvbx_k_inst.h"
namespace tvbx {
Kernel2Fn k2_nosmem(int spc) { TVBX_SPC_SWITCH(spc, false, 8, false, false, false, K2_MAXT, false) }
}  // namespace tvbx
