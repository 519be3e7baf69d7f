// k_sweep_tma for meshes whose memory-contiguous transverse extent is 512 cells (CW = 2 columns per
// chunk, G = 8 chunks per thread, one ray row per warp: the 32 intensity registers of a mirror pair).
// One translation unit per width so that they compile in parallel.
#include "rt_sweep.cuh"

namespace rt {
cudaError_t launch_sweep_nb512(const SweepLaunch &L, cudaStream_t st) { return launch_sweep_nb<2, 8, 1>(L, st); }
int ctas_per_sm_nb512(int rows, int stages, bool pair) { return ctas_per_sm_nb<2, 8, 1>(rows, stages, pair); }
}  // namespace rt
