// lra_degrid_region_ng4.cu -- the region degridder's kernels for passes of 4 grids (lra_degrid_region.cuh).
#include "lra_degrid_region.cuh"

template int lra_degrid_launch_ng<4>(lra_plan*, const lra_region_args&, const lra_geom&, int, cudaStream_t);
