// Internal declarations shared by rt_api.cu (host planner + C ABI) and rt_kernels.cu (sm_100a kernels).
// Not part of the public boundary (include/rt.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace rt {

constexpr int kF = 20;                         // slope quantisation: 2^-20 (reading A4)
constexpr long long kOne = 1ll << kF;
constexpr float kEx2Bias = 4.0e-8f;           // relative correction of ex2.approx (rt_sweep.cuh one_minus_exp)
constexpr float kKappaMin = 8.673617379884035e-19f;   // 2^-60: kappa floor in the packed copy (reading A7)

// Slab program: the traversal of ONE slab for ALL rays of a direction (identical because lattice
// rays differ by whole cells).  Up to three pieces; between pieces the ray steps to the next cell
// along b (SB), along c (SC) or both.  Zero-length pieces are dropped (P bits clear) but their
// step still happens (a ray that lands exactly on a cell boundary at the end of the slab).
struct SlabProg {
    float len0, len1, len2;                    // path lengths in units of length (frac * L * cell_width)
    unsigned flags;
};
enum : unsigned { F_SB1 = 1u, F_SC1 = 2u, F_SB2 = 4u, F_SC2 = 8u, F_P1 = 16u, F_P2 = 32u };
// Above the traversal flags the flags word carries the row shift of the slab, floor(v0 + k m_c) mod Nc (v0 = the
// sub-lattice's offset along c): the memory row of ray row q at slab k is (q + shift) mod Nc.  Extents are <= 2^20.
constexpr unsigned kFlagMask = 63u;
constexpr int kShiftBit = 8;

// Per-direction device record.
struct DirDev {
    long long base;      // element offset (within one bin) of canonical (k=0, l=0), memory column 0
    long long sk, sl;    // signed element strides along canonical k (dominant axis) and l (transverse c)
    int sj;              // +1 / -1: rays move towards higher / lower memory columns
    int Na, Nb, Nc;      // extents along a, b (memory-contiguous axis of the layout), c
    int layout;          // bits 0-3: 0 native [z][y][x], 1 transposed [x][z][y] (x-dominant directions); bits 8-10,
                         // 12-14, 16-18: entry faces along a, b, c (face = 2 * axis + 1 if marching towards -axis)
    int prog_off;        // index of the first SlabProg of this direction
    float invL;          // 1 / (L * cell_width)
    int Mb, Mc;          // quantised slopes (generic kernel recomputes the traversal per ray)
    int sub;             // sub-lattice of an r-rays-per-cell set: alpha | beta << 8 | r << 16 (0 = the r = 1 lattice)
};
static_assert(sizeof(DirDev) == 64, "DirDev layout");

// Offset (in units of 2^-20 cells) of a sub-lattice's rays on the plane a = 0 along b (which = 0) or c (which = 1):
// (2 alpha + 1) / (2 r) (reading O3).  r rays per cell width = r^2 unit lattices with these offsets.
__host__ __device__ __forceinline__ int sub_offset(int sub, int which)
{
    const int r = (sub >> 16) > 0 ? (sub >> 16) : 1;
    const int idx = which ? ((sub >> 8) & 255) : (sub & 255);
    return (2 * idx + 1) * (int)(kOne / (2 * r));
}

// MODE_OWNERS (rt_debug_writer_counts): the J-mode schedule with every accumulator store replaced by an atomic
// increment of the stored-to element, so that the number of writers per cell, accumulator array and launch can be read back
enum Mode : int { MODE_J = 0, MODE_COUNT = 1, MODE_DS = 2, MODE_OWNERS = 3 };

struct SweepLaunch {
    const float2 *P;         // packed (kappa, S) field of the batch's layout, [nbins][cells]
    float *acc;              // slot accumulators of that layout: [slots][nbins][cells]
    float *accC;             // seam accumulators, same shape
    const DirDev *dirs;      // device array of all direction records
    const SlabProg *prog;    // device array of all slab programs
    const int *batch;        // device array: direction index per slot of this launch
    int nslots;              // generic kernel: grid.y = entries of the launch; owned kernel: slots the entries cycle through
    int fresh_below;         // owned kernel, MODE_J: entries below this index are the first users of their slots in the sweep
    int tiles, item0, nitems;// owned kernel: CTAs per entry; first work item and number of work items of this launch (grid.x)
    int nbins;               // grid.z
    long long ncell;
    const float *Ibc;        // device [nbins][6]: inflow per bin and entry face (-x, +x, -y, +y, -z, +z)
    int Nb, Nc;              // common to the batch (same layout => same Nb; Nc may differ per direction)
    int rows;                // rays rows per warp
    int mode;
    int variant;             // generic kernel: 0 = four groups (one launch per group), 1 = atomics
    int group;               // generic kernel: group id 0..3
    int stages;              // owned kernel: depth of the TMA shared-memory ring (2..4)
    int rev;                 // owned kernel, single directions: all slots have a reflected b component (sj < 0)
    int pair;                // owned TMA kernel, MODE_J: every slot carries a direction and its b-mirror (rt_kernels.cu "mirror pairs")
    int pp;                  // P is pair-packed (below)
    int handoff;             // owned kernel: seam partials are handed to the next warp of the CTA in shared memory (ablation)
    int nbp;                 // bins packed per row of P / acc / accC (1: bins are planes; 3: packed_cell below, packed kernel)
};

// Packed-field layouts.  Interleaved: float2 (kappa, S) per cell.  Pair-packed (layouts swept by the
// owned kernel with two columns per chunk): every two adjacent cells of a row are one float4
// (kappa0, kappa1, S0, S1), so that a 16-byte shared-memory load delivers the operands of the packed
// fp32x2 instructions as aligned register pairs.  Index of kappa of cell o in the float view; S is
// at + 1 (interleaved) or + 2 (pair-packed).
__host__ __device__ __forceinline__ size_t field_index(size_t o, int pp) { return pp ? 4 * (o >> 1) + (o & 1) : 2 * o; }
__host__ __device__ __forceinline__ int field_s_offset(int pp) { return pp ? 2 : 1; }

// Offset (in cells) of (bin, row, column) in a packed field or accumulator of one layout.  nbp = 1: bins are planes
// [bin][row][column].  nbp > 1 (multi-bin packed loads): groups of nbp bins share a row, [group][row][bin in group][column],
// so that one bulk copy of a row feeds nbp intensity recurrences.  rows = rows per bin of the layout, pitch = padded row width.
__host__ __device__ __forceinline__ size_t packed_cell(int bin, size_t row, int col, int nbp, int pitch, size_t rows)
{
    return (((size_t)(bin / nbp) * rows + row) * nbp + (size_t)(bin % nbp)) * pitch + col;
}

// launchers (rt_kernels.cu); all return cudaError_t of the launch
cudaError_t launch_build_programs(const DirDev *dirs, int ndirs, int max_na, SlabProg *prog, double cell_width,
                                  const double *Lvals, cudaStream_t st);
cudaError_t launch_pack_fields(const float *kappa, const float *S, float2 *Pnat, float2 *PT, int ppN, int ppT,
                               int nx, int ny, int nz, int nxp, int nyp, int nbins, int nbp, cudaStream_t st);
bool owned_supported(int Nb, int Nc, int rows, int nbp = 1);
int owned_ctas_per_sm(int Nb, int rows, int stages, bool pair, int nbp = 1);
constexpr int kOwnedWarpsPerCta = 4;
constexpr bool kBinpackDefault = false;        // three bins per row by default when eligible (rt_api.cu ensure_buffers)
constexpr int kPackedRows128 = 1;              // ray rows per warp of the packed kernel on 128-cell rows
constexpr int kOverlapWaveDiv = 2;             // overlapped schedule: launches of 1 / kOverlapWaveDiv of a wave (rt_api.cu)
constexpr int kShortRowStages = 2;             // TMA ring depth for rows of <= 64 cells (rt_api.cu stages_for)
cudaError_t launch_sweep_owned(const SweepLaunch &L, cudaStream_t st);
cudaError_t launch_sweep_generic(const SweepLaunch &L, int max_lattice_b, int max_lattice_c, cudaStream_t st);
cudaError_t launch_normalise(float *J, const float2 *Pnat, int ppN, const float *accN, const float *accNC, int slotsN,
                             const float *accT, const float *accTC, int slotsT,
                             int nx, int ny, int nz, int nxp, int nyp, int nbins, int nbp, float inv_nd, int add_S, cudaStream_t st);
cudaError_t launch_rates(float *Gamma, float *Heat, const float2 *Pnat, int ppN, const float *accN, const float *accNC,
                         int slotsN, const float *accT, const float *accTC, int slotsT, int nx, int ny, int nz,
                         int nxp, int nyp, int nbins, int nbp, float inv_nd, const float *w4, cudaStream_t st);
cudaError_t launch_combine(float *J, const float *sum, const float2 *Pnat, int ppN, int nx, int ny, int nz, int nxp,
                           int nbins, int nbp, float inv_nd, int add_S, cudaStream_t st);
cudaError_t launch_point_sources(float *Q, float *tau_out, const float2 *Pnat, int ppN, int nx, int ny, int nz, int nxp,
                                 const int *src_dev, const float *lum_dev, int nsrc, int nbins, int nbp, float cell_width,
                                 int diag_src, int diag_bin, unsigned long long *steps_dev, cudaStream_t st);
// weights of the per-species point-source rates (rt_point_source_rates, eqs. A5-A6): wG = 1 / h nu_b, wH = (h nu_b - h nu_i) / h nu_b
// for bins at or above the species' threshold, 0 below it
constexpr int kMaxSpecies = 8;
struct SpeciesWeights { float wG[kMaxSpecies][16], wH[kMaxSpecies][16]; };
cudaError_t launch_point_source_rates(float *Gamma, float *Heat, const float *Q, const float *ksp, const float *nsp,
                                      const float2 *Pnat, int ppN, int nx, int ny, int nz, int nxp, int nbins, int nbp,
                                      int nspecies, const SpeciesWeights &W, int sm_count, cudaStream_t st);
cudaError_t launch_counts_finalise(unsigned *counts, const float *accN, const float *accNC, int slotsN,
                                   const float *accT, const float *accTC, int slotsT,
                                   int nx, int ny, int nz, int nxp, int nyp, cudaStream_t st);
// per-cell sum of ds of ONE direction held in slot 0 of the given layout: writes {sum, min, max} (fp64)
cudaError_t launch_ds_reduce(double *out3, const float *acc, const float *accC, long long ncell, int pitch, int width,
                             cudaStream_t st);
cudaError_t launch_sum_u32(unsigned long long *out, const unsigned *counts, long long n, cudaStream_t st);
// writer counts of one launch in MODE_OWNERS: out2[0] = max(out2[0], max_i w[i]), out2[1] += sum_i w[i] over n floats
cudaError_t launch_owner_reduce(unsigned long long *out2, const float *w, long long n, cudaStream_t st);

// records the text of a CUDA error for rt_last_cuda_error() and returns RT_ECUDA (rt_api.cu; for rt_static.cu)
int api_cuda_fail(cudaError_t e);

// `reps` passes of the streaming probe over n4 float4 in one launch (rmw = 0: read, 1: read-modify-write)
cudaError_t launch_probe(float4 *buf, size_t n4, int rmw, int reps, int sm_count, cudaStream_t st);

}  // namespace rt
