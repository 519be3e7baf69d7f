// k_sweep_tma for meshes whose memory-contiguous transverse extent is 32 cells (CW = 1 columns per
// chunk, G = 1 chunks per thread).  One translation unit per width so that they compile in parallel.
#include "rt_sweep.cuh"

namespace rt {
cudaError_t launch_sweep_nb32(const SweepLaunch &L, cudaStream_t st) { return launch_sweep_nb<1, 1>(L, st); }
int ctas_per_sm_nb32(int rows, int stages, bool pair) { return ctas_per_sm_nb<1, 1>(rows, stages, pair); }
}  // namespace rt
