// k_grid_step instantiations for interpolation order 4 (see vfps_launch.h)
#include "vfps_grid.cuh"
#include "vfps_launch.h"

namespace vfps {

const void *grid_kernel_o4(bool manh, bool clamp)
{
    if (clamp) return manh ? (const void *)k_grid_step<4, true, true> : (const void *)k_grid_step<4, false, true>;
    return manh ? (const void *)k_grid_step<4, true, false> : (const void *)k_grid_step<4, false, false>;
}

}  // namespace vfps
