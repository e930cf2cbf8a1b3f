// tvbx_k_inst.h -- switch over the compile-time simulations per CTA of an integrate2_kernel instance family
#pragma once
#include "tvbx_kernels.h"
#define TVBX_SPC_SWITCH(spc, ...)                                   \
  switch (spc) {                                                    \
    case 1: return integrate2_kernel<1, __VA_ARGS__>;               \
    case 2: return integrate2_kernel<2, __VA_ARGS__>;               \
    case 3: return integrate2_kernel<3, __VA_ARGS__>;               \
    case 4: return integrate2_kernel<4, __VA_ARGS__>;               \
    case 5: return integrate2_kernel<5, __VA_ARGS__>;               \
    case 6: return integrate2_kernel<6, __VA_ARGS__>;               \
    case 7: return integrate2_kernel<7, __VA_ARGS__>;               \
    default: return integrate2_kernel<8, __VA_ARGS__>;              \
  }
