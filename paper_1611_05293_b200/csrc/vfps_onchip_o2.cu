// k_onchip_step instantiations for interpolation order 2 (see vfps_launch.h)
#include "vfps_onchip.cuh"
#include "vfps_launch.h"

namespace vfps {

const void *onchip_kernel_o2(int N, bool tab, bool clamp)
{
    (void)clamp;          // linear interpolation never leaves the interval of its two nodes: the clamp is the identity
#define VFPS_OC(NN) (tab ? (const void *)k_onchip_step<2, NN, true> : (const void *)k_onchip_step<2, NN, false>)
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
