// lra_grid_region_ng4.cu -- the region gridder's kernels for passes of 4 grids (lra_grid_region.cuh).
#include "lra_grid_region.cuh"

template int lra_grid_launch_ng<4>(lra_plan*, const lra_region_args&, const lra_geom&, int, cudaStream_t);
