// tvbx_kernels.cu -- which integrate2_kernel instance serves a launch (host only; the instances are in tvbx_k_*.cu)
#include "tvbx_kernels.h"
namespace tvbx {
Kernel2Fn pick_kernel2(const Kernel2Key& k) {
  if (k.ws && k.grp) return k2_wsg(k.spc);
  if (k.ws) return k2_ws(k.spc, k.sring);
  if (k.sring && k.gce == 1) return k2_g1(k.spc);
  if (k.sring) return k.gce == 2 ? k2_g2(k.spc, true) : (k.gce == 4 ? k2_g4(k.spc, true) : k2_g8_small_sring(k.spc));
  if (k.clu && k.vec) return k2_vec(k.spc, k.smemtab);
  if (k.clu) return (k.small && k.smemtab && k.gce == 8) ? k2_clu_small(k.spc) : k2_clu(k.spc);
  if (!k.smemtab) return k2_nosmem(k.spc);
  if (k.gce == 2) return k2_g2(k.spc, false);
  if (k.gce == 4) return k2_g4(k.spc, false);
  return k.small ? k2_g8_small(k.spc, k.isamp) : k2_g8(k.spc, k.isamp);
}
}  // namespace tvbx
