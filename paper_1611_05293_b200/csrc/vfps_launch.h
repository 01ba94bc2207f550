// vfps_launch.h -- kernel look-up between the translation units of libvfps.so.
//
// The persistent engines instantiate dozens of kernel templates (grid size x interpolation order
// x variant).  Each family lives in its own .cu files (one per interpolation order) so that
// build.py compiles them in parallel; vfps_api.cu launches them through cudaLaunchKernelExC /
// cudaLaunchCooperativeKernel with the pointers returned here.  nullptr = not instantiated.
#pragma once

namespace vfps {

// k_onchip_step<ORDER, N, TAB, CLAMP> (vfps_onchip.cuh); N in {64, 128, 256, 512}
const void *onchip_kernel_o2(int N, bool tab, bool clamp);
const void *onchip_kernel_o3(int N, bool tab, bool clamp);
const void *onchip_kernel_o4(int N, bool tab, bool clamp);

// k_cluster_step<ORDER, N, MANH> (vfps_cluster.cuh); N in {32, 64, 128, 256, 512}
const void *cluster_kernel_o2(int N, bool manh);
const void *cluster_kernel_o3(int N, bool manh);
const void *cluster_kernel_o4(int N, bool manh);

// k_grid_step<ORDER, MANH, CLAMP> (vfps_grid.cuh)
const void *grid_kernel_o2(bool manh, bool clamp);
const void *grid_kernel_o3(bool manh, bool clamp);
const void *grid_kernel_o4(bool manh, bool clamp);

// k_grid2_step<ORDER, CLAMP> (vfps_grid2.cuh); arguments (GridConst, Grid2Args, CUtensorMap)
const void *grid2_kernel_o2(bool clamp);
const void *grid2_kernel_o3(bool clamp);
const void *grid2_kernel_o4(bool clamp);

}  // namespace vfps
