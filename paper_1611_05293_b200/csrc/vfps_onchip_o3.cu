// k_onchip_step instantiations for interpolation order 3 (see vfps_launch.h)
#include "vfps_onchip.cuh"
#include "vfps_launch.h"

namespace vfps {

const void *onchip_kernel_o3(int N, bool tab, bool clamp)
{
#define VFPS_OC(NN)                                                                                     \
    (clamp ? (tab ? (const void *)k_onchip_step<3, NN, true, true> : (const void *)k_onchip_step<3, NN, false, true>)  \
           : (tab ? (const void *)k_onchip_step<3, NN, true, false> : (const void *)k_onchip_step<3, NN, false, false>))
    switch (N) {
        case 64: return VFPS_OC(64);
        case 128: return VFPS_OC(128);
        case 256: return VFPS_OC(256);
        case 512: return VFPS_OC(512);
        default: return nullptr;
    }
#undef VFPS_OC
}

}  // namespace vfps
