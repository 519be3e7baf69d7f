// k_sweep_tma for meshes whose memory-contiguous transverse extent is 256 cells (CW = 2 columns per
// chunk, G = 4 chunks per thread).  One translation unit per width so that they compile in parallel.
#include "rt_sweep.cuh"

namespace rt {
cudaError_t launch_sweep_nb256(const SweepLaunch &L, cudaStream_t st) { return launch_sweep_nb<2, 4>(L, st); }
int ctas_per_sm_nb256(int rows, int stages, bool pair) { return ctas_per_sm_nb<2, 4>(rows, stages, pair); }
}  // namespace rt
