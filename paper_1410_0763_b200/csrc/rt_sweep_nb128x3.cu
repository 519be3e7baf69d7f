// k_sweep_tma with three frequency bins packed per row (multi-bin packed loads, eqs. 22-23) for
// rows of 128 cells: CW = 2 column(s) per chunk, G = 6 chunks per thread = 3 bins x 2 chunk(s).
// One translation unit per width so that they compile in parallel.
#include "rt_sweep.cuh"

namespace rt {
cudaError_t launch_sweep_nb128x3(const SweepLaunch &L, cudaStream_t st) { return launch_sweep_packed<2, 6, 3>(L, st); }
int ctas_per_sm_nb128x3(int rows, bool pair) { return ctas_per_sm_packed<2, 6, 3>(rows, pair); }
}  // namespace rt
