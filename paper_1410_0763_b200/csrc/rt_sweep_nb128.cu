// k_sweep_tma for meshes whose memory-contiguous transverse extent is 128 cells (CW = 2 columns per
// chunk, G = 2 chunks per thread).  One translation unit per width so that they compile in parallel.
#include "rt_sweep.cuh"

namespace rt {
cudaError_t launch_sweep_nb128(const SweepLaunch &L, cudaStream_t st) { return launch_sweep_nb<2, 2>(L, st); }
int ctas_per_sm_nb128(int rows, int stages, bool pair) { return ctas_per_sm_nb<2, 2>(rows, stages, pair); }
}  // namespace rt
