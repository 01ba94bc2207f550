// k_cluster_step instantiations for interpolation order 4 (see vfps_launch.h)
#include "vfps_cluster.cuh"
#include "vfps_launch.h"

namespace vfps {

const void *cluster_kernel_o4(int N, bool manh)
{
#define VFPS_CL(NN) (manh ? (const void *)k_cluster_step<4, NN, true> : (const void *)k_cluster_step<4, NN, false>)
    switch (N) {
        case 32: return VFPS_CL(32);
        case 64: return VFPS_CL(64);
        case 128: return VFPS_CL(128);
        case 256: return VFPS_CL(256);
        case 512: return VFPS_CL(512);
        default: return nullptr;
    }
#undef VFPS_CL
}

}  // namespace vfps
