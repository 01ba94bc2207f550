// k_grid2_step instantiations for interpolation order 4 (see vfps_launch.h)
#include "vfps_grid2.cuh"
#include "vfps_launch.h"

namespace vfps {

const void *grid2_kernel_o4(bool clamp)
{
    return clamp ? (const void *)k_grid2_step<4, true> : (const void *)k_grid2_step<4, false>;
}

}  // namespace vfps
