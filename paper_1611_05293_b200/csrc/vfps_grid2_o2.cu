// k_grid2_step instantiations for interpolation order 2 (see vfps_launch.h)
#include "vfps_grid2.cuh"
#include "vfps_launch.h"

namespace vfps {

const void *grid2_kernel_o2(bool clamp)
{
    return clamp ? (const void *)k_grid2_step<2, true> : (const void *)k_grid2_step<2, false>;
}

}  // namespace vfps
