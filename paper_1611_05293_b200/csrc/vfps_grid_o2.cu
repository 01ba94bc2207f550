// k_grid_step instantiations for interpolation order 2 (see vfps_launch.h)
#include "vfps_grid.cuh"
#include "vfps_launch.h"

namespace vfps {

const void *grid_kernel_o2(bool manh, bool clamp)
{
    if (clamp) return manh ? (const void *)k_grid_step<2, true, true> : (const void *)k_grid_step<2, false, true>;
    return manh ? (const void *)k_grid_step<2, true, false> : (const void *)k_grid_step<2, false, false>;
}

}  // namespace vfps
