// lra_grid_region_ng1.cu -- the region gridder's kernels for passes of 1 grid (lra_grid_region.cuh).
#include "lra_grid_region.cuh"

template int lra_grid_launch_ng<1>(lra_plan*, const lra_region_args&, const lra_geom&, int, cudaStream_t);
