/*
 * rt.h -- C ABI of the B200-native diffuse-radiation ray sweep (arXiv:1410.0763, Tanaka et al.).
 *
 * The library computes, for a uniform 3-D mesh with absorption coefficient kappa and source
 * function S per cell and a set of N_d directions, the mean intensity
 *
 *     J_in = (1/N_d) sum_i  Ibar^{ave,in}(n_i)        (eq. 13)
 *     J    = J_in + S                                 (eq. 12)
 *
 * where, per direction, equally spaced parallel rays (one per cell cross-section on the
 * plane normal to the dominant axis) are marched cell by cell with
 *
 *     I_out = I_in exp(-dtau) + S (1 - exp(-dtau)),  dtau = kappa * ds      (eq. 7)
 *     Ibar_in = I_in (1 - exp(-dtau)) / dtau                                (eq. 8)
 *     Ibar^{ave,in} = sum_j dtau_j Ibar_in,j / sum_j dtau_j                 (eqs. 10-11)
 *
 * and concurrently marching rays never write the same cell (section 3.1); here
 * that is achieved by cell ownership instead of the paper's four sequential ray groups.
 *
 * Conventions
 *  - Every call returns RT_OK (0) or a negative RT_E* code; nothing throws, aborts or prints.
 *  - "host" / "device" is stated for every pointer.  Device pointers must belong to the CUDA
 *    device that was current when rt_create was called; every call makes that device current for
 *    its duration and restores the caller's.
 *  - Field arrays are fp32, C-contiguous [nbins][nz][ny][nx] (x fastest).
 *  - `cuda_stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  All device
 *    work is enqueued on it; calls are asynchronous unless stated otherwise.
 *  - The context owns all internal device memory; the caller owns kappa, S, J and count buffers.
 *  - One context must not be used from two host threads at once; different contexts are independent.
 *  - The library has no CPU fallback: without a usable CUDA device rt_create fails with RT_ECUDA.
 */
#ifndef RT_H_
#define RT_H_

#ifdef __cplusplus
extern "C" {
#endif

typedef struct rt_ctx rt_ctx;

/* error codes */
#define RT_OK        0
#define RT_EINVAL   -1   /* bad argument: null pointer, non-positive dims, zero direction vector, unsupported option */
#define RT_ENOMEM   -2   /* host or device allocation failed */
#define RT_ECUDA    -3   /* CUDA runtime error; text via rt_last_cuda_error() */
#define RT_ESTATE   -4   /* call order: e.g. rt_sweep before rt_set_fields */
#define RT_ELIMIT   -5   /* size beyond the fixed capacity of an entry point that never allocates (RT_STATIC_MAX_*) */

/* rt_create flags */
#define RT_OWNED            0u   /* default: atomic-free, one writer per cell (ownership + seam accumulators) */
#define RT_ATOMIC_ABLATION  1u   /* ablation: every ray segment does atomicAdd into the accumulator */
#define RT_PAPER_GROUPS     2u   /* ablation: the paper's four sequential ray groups with plain stores */

/* rt_sweep `what` */
#define RT_J_IN     0u           /* eq. 13 */
#define RT_J_TOTAL  1u           /* eq. 12: J_in + S */
#define RT_SUM_IN   2u           /* N_d * J_in of this context's directions: the un-normalised sum of eq. 13 (for rt_combine) */

/*
 * HEALPix ring-scheme pixel centres (Gorski et al. 2005, cited at PAPER.md:183, 463).
 *   nside     : resolution parameter >= 1
 *   dirs_out  : HOST, fp64 [12*nside*nside][3], unit vectors, RING order (north to south)
 * Returns the number of directions written, or RT_EINVAL.
 */
int rt_healpix_dirs(int nside, double *dirs_out);

/*
 * Create a sweep context: quantise the directions (dominant axis, reflections, slopes in units of
 * 2^-20, slab length), build the per-direction slab programs on the device (the integer traversal
 * of PAPER.md:86 / Fig. 2, identical for every ray of a direction), choose layouts, allocate.
 *   out           : HOST, receives the context
 *   nx, ny, nz    : mesh dimensions (x fastest)
 *   nbins         : frequency bins sharing one geometry (eq. 22), 1..16
 *   dirs, ndirs   : HOST, fp64 [ndirs][3], need not be normalised, none may be zero; copied
 *   rays_per_cell : r = rays per cell width in each transverse axis, i.e. ray spacing = dH / r;
 *                   a power of two, 1..16 (RT_EINVAL otherwise).  r > 1 is swept as r^2 interleaved unit lattices
 *                   with offsets (2 alpha + 1)/(2 r), each with its own slab program; per cell and direction
 *                   sum ds = r^2 L, which the normalisation accounts for.  Cost and segment counts scale with r^2.
 *   cell_width    : mesh spacing dH (> 0); kappa is per unit length, so dtau = kappa * ds * dH
 *   flags         : RT_OWNED | RT_ATOMIC_ABLATION | RT_PAPER_GROUPS
 * Limits (RT_EINVAL beyond): each dimension <= 2^20, nx*ny*nz < 2^31, 3 * ndirs * r^2 < 2^24 (per-cell segment
 * counts stay exact in the fp32 accumulators).
 * Synchronises the device once (table build).  Returns RT_OK / RT_EINVAL / RT_ENOMEM / RT_ECUDA.
 */
int rt_create(rt_ctx **out, int nx, int ny, int nz, int nbins,
              const double *dirs, int ndirs, int rays_per_cell, double cell_width, unsigned flags);

/*
 * Set the medium.  Enqueues a repack of (kappa, S) into the packed sweep layouts on `cuda_stream`.
 *   kappa_dev, S_dev : DEVICE, fp32 [nbins][nz][ny][nx]; borrowed only until the enqueued repack
 *                      has completed on the stream; the library keeps its own packed copies.
 * kappa must be >= 0 and finite; kappa = 0 is allowed (f(0) = 1, reading A7).
 */
int rt_set_fields(rt_ctx *ctx, const float *kappa_dev, const float *S_dev, void *cuda_stream);

/*
 * Boundary inflow intensity per bin (default 0; the diffuse field has no external source in the
 * paper's tests).   I_bc_host : HOST, fp32 [nbins].
 * Synchronises the device (sweeps in flight on any stream keep the old values), then copies.
 */
int rt_set_inflow(rt_ctx *ctx, const float *I_bc_host);

/*
 * Boundary inflow per bin and entry face (boundary illumination as in the paper's Test 3).
 *   I_face_host : HOST, fp32 [nbins][6], faces in the order -x, +x, -y, +y, -z, +z, each >= 0 and finite.
 * A ray starts with the value of the face through which it enters the box, i.e. the face it crosses last: a
 * ray marching towards +x that starts inside the transverse extent enters through -x; one that comes in from
 * the side enters through that side face; through an edge (both side planes at once): the c-axis face
 * (reading A10).  rt_set_inflow(v) is the same as all six faces = v.  Synchronises the device, then copies.
 */
int rt_set_inflow_faces(rt_ctx *ctx, const float *I_face_host);

/*
 * The same two updates without the device-wide synchronisation: enqueued on `cuda_stream` like every other call, for a
 * boundary illumination that changes every iteration next to work on other streams.  The values
 * travel in the parameters of a one-block kernel (no staging buffer): the host array may be reused as soon as the call
 * returns.  Ordering is the stream's: sweeps enqueued later on `cuda_stream` (CUDA-graph replays included) use the new
 * values, sweeps enqueued earlier on it the old ones; with respect to sweeps of this context on OTHER streams the
 * caller orders the update with events, as for any device buffer.  Arguments and value checks as above.
 */
int rt_set_inflow_async(rt_ctx *ctx, const float *I_bc_host, void *cuda_stream);
int rt_set_inflow_faces_async(rt_ctx *ctx, const float *I_face_host, void *cuda_stream);

/*
 * One full sweep over all directions ("one iteration" of PAPER.md:322).
 *   J_dev : DEVICE, fp32 [nbins][nz][ny][nx], caller-owned, fully overwritten
 *   what  : RT_J_IN, RT_J_TOTAL or RT_SUM_IN
 * Asynchronous on `cuda_stream`.  RT_ESTATE if rt_set_fields has not been called.
 */
int rt_sweep(rt_ctx *ctx, float *J_dev, unsigned what, void *cuda_stream);

/*
 * Combine step of a direction-sharded sweep, the paper's multi-accelerator scheme (every
 * device holds the whole mesh and a share of the directions; the partial mean intensities are summed).  Each
 * shard is a context created with its own directions and swept with RT_SUM_IN; the caller adds the shards'
 * results element-wise (one all-reduce(sum), e.g. NCCL through torch.distributed) and then calls
 *     J_in = sum / ndirs_total (eq. 13),   J = J_in + S (eq. 12)
 *   sum_dev     : DEVICE, fp32 [nbins][nz][ny][nx], the added RT_SUM_IN results of all shards
 *   ndirs_total : number of directions of the whole set
 *   what        : RT_J_IN or RT_J_TOTAL
 *   J_dev       : DEVICE, fp32 [nbins][nz][ny][nx], fully overwritten; may alias sum_dev
 * Asynchronous on `cuda_stream`.  RT_ESTATE if rt_set_fields has not been called (S comes from the packed fields).
 */
int rt_combine(rt_ctx *ctx, const float *sum_dev, long long ndirs_total, unsigned what, float *J_dev, void *cuda_stream);

/*
 * One full sweep followed by the rates epilogue instead of J: the photo-ionisation and photo-heating
 * rates of the diffuse field (eqs. 14-15) for a spectrum of rectangular bins
 * (eqs. 22-23), per cell
 *     Gamma = sum_b  wG[b] * J_in[b] + lG[b] * S[b]
 *     Heat  = sum_b  wH[b] * J_in[b] + lH[b] * S[b]
 * with caller-supplied per-bin weights ("estimated prior to the simulations"):
 *     wG[b] = 4 pi int_bin sigma/(h nu) dnu,  wH[b] = 4 pi int_bin sigma (1 - nu_i/nu) dnu   (J_in flat in the bin, eq. 19)
 *     lG[b], lH[b] = the same integrals weighted by S_nu / S[b] (the source function's shape inside the bin).
 * With one bin, S of eq. 18 and its shape in lG, lH this is eqs. 20-21: lG*S is the local
 * term  delta_alpha n_e n_HII / n_HI.  Passing lG = wG, lH = wH gives eq. 14-15 applied to J = J_in + S.
 *   Gamma_dev, Heat_dev : DEVICE, fp32 [nz][ny][nx], caller-owned, fully overwritten
 *   wG, lG, wH, lH      : HOST, fp64 [nbins] (converted to fp32), finite
 * Asynchronous on `cuda_stream`.  RT_ESTATE if rt_set_fields has not been called.
 */
int rt_sweep_rates(rt_ctx *ctx, float *Gamma_dev, float *Heat_dev, const double *wG, const double *lG,
                   const double *wH, const double *lH, void *cuda_stream);

/*
 * RT from point radiation sources (section 2.1) with the photon-conserving estimate of
 * Appendix 1: one light-ray per (source, cell) from the source through the cell centre
 * (long characteristics; cost N_m^(4/3) per source).  With tau the optical depth of the cells
 * crossed before the target cell, r_in / r_out the distances at which the ray enters / leaves the target cell
 * and dtau = kappa_cell (r_out - r_in), per cell and bin
 *     Q = sum_alpha  L[alpha][bin] exp(-tau) (1 - exp(-dtau)) / (4 pi/3 (r_out^3 - r_in^3))       (eqs. A1-A3 / shell volume)
 * i.e. the absorption rate per unit volume; eq. A5's rate of species i is Q (dtau_i/dtau) / (n_i h nu).
 * Uses the kappa of the last rt_set_fields (S is not used).  Lengths are in units of cell_width.
 *   src_fix_host : HOST, int32 [nsrc][3], source positions in units of 1/256 cell width (0 .. 256*dim), so that
 *                  the traversal is exact; a source on a cell boundary belongs to the cell a ray moves into; the
 *                  cell whose centre IS the source uses r_in = 0, r_out = cell_width/2
 *   lum_host     : HOST, fp64 [nsrc][nbins] luminosities (>= 0, converted to fp32)
 *   Q_dev        : DEVICE, fp32 [nbins][nz][ny][nx], fully overwritten
 *   tau_dev      : DEVICE, fp32 [nz][ny][nx] or NULL: tau of source diag_src in bin diag_bin (diagnostic)
 *   steps_host   : HOST or NULL: number of positive-length ray pieces marched per bin, all sources (integer
 *                  traversal data for the parity gate)
 * Mesh dimensions must be <= 1024 (RT_EINVAL).  Asynchronous on `cuda_stream`: the source tables are copied into
 * context-owned device tables through a pinned staging buffer (only when they differ from the previous call's), the
 * host arrays may be reused as soon as the call returns.  Only a call with steps_host != NULL synchronises the stream.
 */
int rt_point_sources(rt_ctx *ctx, const int *src_fix_host, const double *lum_host, int nsrc, float *Q_dev,
                     int diag_src, int diag_bin, float *tau_dev, unsigned long long *steps_host, void *cuda_stream);

/*
 * Per-species photo-ionisation and photo-heating rates from the point-source absorption rate (Appendix 1,
 * PAPER.md:378-388, eqs. A4-A6), as an elementwise epilogue of rt_point_sources.  With Q_b the absorbed
 * energy per unit time and shell volume in bin b (rt_point_sources), kappa_b the total opacity of the cell
 * (the kappa of the last rt_set_fields), kappa_i,b the part of it contributed by species i, n_i the number
 * density of species i and h nu_b the photon energy of bin b:
 *     Gamma_i = (1/n_i) sum_{b: h nu_b >= h nu_i}  (kappa_i,b / kappa_b)  Q_b / (h nu_b)                    (A4, A5)
 *     Heat_i  = (1/n_i) sum_{b: h nu_b >= h nu_i}  (kappa_i,b / kappa_b)  Q_b (h nu_b - h nu_i) / (h nu_b)  (A6)
 * (dtau_i / dtau = kappa_i / kappa inside one cell; N_i = n_i x shell volume, and Q is already per unit shell
 * volume; the frequency integrals are sums over the rectangular bins of eqs. 22-23.  Eq. A6 is read with the
 * species' own absorption rate, like eq. 6: DESIGN.md reading PS-f.)  A cell with n_i <= 0 gets 0.
 *   Q_dev        : DEVICE, fp32 [nbins][nz][ny][nx] (output of rt_point_sources)
 *   kappa_sp_dev : DEVICE, fp32 [nspecies][nbins][nz][ny][nx], opacity contributed by each species (>= 0)
 *   n_sp_dev     : DEVICE, fp32 [nspecies][nz][ny][nx], number densities
 *   hnu_host     : HOST, fp64 [nbins], photon energy of each bin (> 0)
 *   hnu_thr_host : HOST, fp64 [nspecies], threshold energy h nu_i of each species (>= 0)
 *   Gamma_dev, Heat_dev : DEVICE, fp32 [nspecies][nz][ny][nx], fully overwritten
 * 1 <= nspecies <= 8 (RT_EINVAL otherwise).  Asynchronous on `cuda_stream`; RT_ESTATE before rt_set_fields.
 */
int rt_point_source_rates(rt_ctx *ctx, const float *Q_dev, const float *kappa_sp_dev, const float *n_sp_dev, int nspecies,
                          const double *hnu_host, const double *hnu_thr_host, float *Gamma_dev, float *Heat_dev,
                          void *cuda_stream);

/*
 * rt_point_sources for callers that cannot allocate device memory: no context, no cudaMalloc / cudaFree /
 * cudaMallocHost, no allocating library routine, on any call.
 *
 * Who needs it: a simulation code that claimed (nearly) all of the GPU's memory for its own arena at start-up, code
 * running under a framework's caching allocator, a GPU shared through MPS with a per-client memory limit, or the
 * inside of a time step where the device-wide synchronisation of cudaMalloc / cudaFree would stall the other streams.
 * For them rt_create + rt_set_fields + rt_point_sources is unusable: those allocate tables, packed copies of the
 * fields and a pinned staging buffer.  Here the caller passes kappa and the outputs, and the only other memory the
 * kernel needs -- a device copy of the source tables and the counter of marched ray pieces -- is a fixed array of
 * 143,616 bytes inside the library image (a file-scope __device__ array in csrc/rt_static.cu).  Every GPU on which
 * the process uses this library holds that array from the moment the library's code is loaded there until exit.
 *
 * Same operation, argument meaning and units as rt_point_sources (eqs. A1-A3), except:
 *   nx, ny, nz, nbins, cell_width : the mesh (each dimension <= 1024, nx*ny*nz < 2^31), as rt_create would take them
 *   kappa_dev : DEVICE, fp32 [nbins][nz][ny][nx], read in place (kappa below 2^-60 counts as 2^-60, as in the packed copy);
 *               must stay valid and unchanged until the enqueued kernel has run
 *   src_fix_host, lum_host, nsrc, Q_dev, diag_src, diag_bin, tau_dev, steps_host : as rt_point_sources
 * Capacity: nsrc <= RT_STATIC_MAX_SOURCES and nbins <= RT_STATIC_MAX_BINS; larger -> RT_ELIMIT and nothing is
 * enqueued (use rt_point_sources, or split the sources over several calls and add the Q arrays).
 * Device: the CUDA device current at the call; the pointers must belong to it.
 * First call on a device: looks up the device address of the array (cudaGetSymbolAddress; this is also when the CUDA
 * runtime loads the kernel's module on that device).  Make this first call before any stream capture begins.
 * Sharing: all calls on a device use the one array.  Each call clears the counter and overwrites the tables on
 * `cuda_stream`, so the array never carries state from one call into the next, but two calls whose GPU work overlaps
 * (different streams without an event between them, or two host threads) race on it and give undefined Q.
 * Asynchronous on `cuda_stream` apart from the staging of the two small pageable host tables (they may be reused when
 * the call returns); a call with steps_host != NULL synchronises the stream.
 */
#define RT_STATIC_MAX_SOURCES 1024
#define RT_STATIC_MAX_BINS    16
int rt_point_sources_static(int nx, int ny, int nz, int nbins, double cell_width, const float *kappa_dev,
                            const int *src_fix_host, const double *lum_host, int nsrc, float *Q_dev,
                            int diag_src, int diag_bin, float *tau_dev, unsigned long long *steps_host, void *cuda_stream);

/*
 * Diagnostics required by the parity gates (integer traversal data, summed ds).  They run the same
 * traversal kernel as rt_sweep with the transfer arithmetic replaced by counting.
 *
 * rt_segment_counts: per-cell number of positive-length ray segments.
 *   dir_index  : 0..ndirs-1 for one direction, -1 for the sum over all directions
 *   counts_dev : DEVICE, uint32 [nz][ny][nx], fully overwritten.  Asynchronous.
 * rt_sum_ds: fp32-path sum of segment lengths per direction, widened to fp64.
 *   sum_ds_host : HOST, fp64 [ndirs].  Synchronises the stream.
 *   min_ds_host, max_ds_host : HOST, fp64 [ndirs] or NULL: min / max over cells of the per-cell sum of ds.
 * rt_total_segments: exact total over directions and cells (numerator of the throughput metric,
 *   per bin).  n_host : HOST.  The first call runs a counting traversal and synchronises the stream; the
 *   geometry of a context never changes, so later calls return the cached value.
 */
int rt_segment_counts(rt_ctx *ctx, int dir_index, unsigned int *counts_dev, void *cuda_stream);
int rt_sum_ds(rt_ctx *ctx, double *sum_ds_host, double *min_ds_host, double *max_ds_host, void *cuda_stream);
int rt_total_segments(rt_ctx *ctx, unsigned long long *n_host, void *cuda_stream);

/*
 * Writer-count check of the ownership scheme that replaces the paper's ray groups (section 3.1:
 * "light-rays in each group do not traverse any mesh grid more than once").  Runs the launches of rt_sweep (same
 * work-item ranges, slots, mirror pairs, rows per warp, handoff) with every accumulator store replaced by an atomic
 * increment of the element it would have written, one launch at a time, and reads the counts back.
 *   out_host : HOST, unsigned long long [8] =
 *     [0] largest number of stores any element of a slot accumulator received within one launch (must be 1)
 *     [1] stores to the slot accumulators, all launches     [2], [3] the same for the seam accumulators ([2] <= 1)
 *     [4] launches checked                                  [5] launches that start or end inside an entry
 *     [6] (entries) x (cells of the entry's padded layout) x nbins: every such element is stored exactly once per
 *         entry, so [1] must equal [6]                      [7] entries (directions or mirror pairs) swept
 * RT_EINVAL unless the context was created with RT_OWNED and every layout runs on the owned kernel.
 * Diagnostic: slow (clears and reduces all slot accumulators around every launch); synchronises the stream.
 */
int rt_debug_writer_counts(rt_ctx *ctx, unsigned long long *out_host, void *cuda_stream);

/*
 * Per-direction record as quantised by the library (for cross-checks against the oracle).
 *   rec_host : HOST, long long [ndirs][6] = {dominant axis, reflect_x | reflect_y<<1 | reflect_z<<2,
 *              M_b, M_c, kernel path (0 = owned fast path, 1 = generic), rays_per_cell}
 *   L_host   : HOST, fp64 [ndirs] slab length in cell widths, or NULL
 */
int rt_direction_records(rt_ctx *ctx, long long *rec_host, double *L_host);

/*
 * Tuning knobs (experiments and ablations; defaults are chosen by rt_create).
 *   "slots"  : concurrent direction slots per launch (each has private accumulators)
 *   "rows"   : rays rows per warp in the owned kernel (1, 2 or 4; 4 only for rows of <= 128 cells; default by row width:
 *              1 up to 64 cells, 4 for 128, 2 for 256, 1 for 512; rows of nx (ny) cells are padded to the next of
 *              32/64/128/256/512, wider ones run on the generic kernel)
 *   "stages" : depth of the owned kernel's TMA shared-memory ring (2 or 3; 4 for rows of <= 64 cells)
 *   "overlap": 1 = every class of directions (layout, dominant axis, pairs / singles, march sense) gets its own slot
 *              range and runs on an internal stream of its own, forked from and joined into the caller's stream, so that
 *              consecutive classes overlap; 0 = one launch after the other; default: 1 when the packed fields fit in
 *              half the L2 (32^3 ... 128^3), else 0
 *   "graph"  : 1 = from its second use on, a (J buffer, what) combination of rt_sweep is replayed as one CUDA graph;
 *              default: only for sweeps of at most two waves of CTAs (launch-latency bound, e.g. 32^3 x 48)
 *   "pair"   : 1 (default) = a direction and its mirror image along the memory-contiguous transverse axis
 *              are marched by the same warp (shared loads, stores and exponentials); 0 = one direction per warp
 *   "handoff": 1 = a warp's seam partial is handed to the next warp of its CTA through a ring in shared memory
 *              instead of the seam accumulator (15 % less DRAM traffic, measured 7 % slower; default 0)
 * Returns RT_EINVAL for unknown keys or unsupported values.  Must be called before rt_set_fields.
 */
int rt_tune(rt_ctx *ctx, const char *key, int value);

/*
 * Device memory the sweep streams through: packed fields of both layouts + slot and seam accumulators (allocates
 * them if that has not happened yet).  bytes_host : HOST.  Used to say whether a workload is L2-resident.
 */
int rt_working_set_bytes(rt_ctx *ctx, unsigned long long *bytes_host);

/*
 * Streaming bandwidth probe of the current device: the denominators of the memory-side roofline that
 * MEASURED_PEAKS.json does not carry ("L2 peak ... the builder must measure it").  One kernel of
 * 8 CTAs per SM x 512 threads streams a zeroed scratch buffer of `bytes` with 16-byte cache-global accesses (about
 * 8 GB of them per timed launch, i.e. many passes over a small buffer):
 *   mode 0 : read only;  mode 1 : read-modify-write of every element (bytes counted twice: read + write)
 * A buffer well below the L2 capacity (<= 64 MB of 126 MB) measures L2, one of >= 1 GB measures HBM.
 *   bytes    : 2^20 .. 2^36;  iters : timed repetitions after two warm-up passes (best is reported)
 *   gbs_host : HOST, GB/s (1e9 bytes per second)
 * Allocates and frees its scratch buffer; synchronises the stream.  Needs no context.
 */
int rt_probe_bandwidth(unsigned long long bytes, int mode, int iters, double *gbs_host, void *cuda_stream);

/* Number of kernel launches issued by the last rt_sweep of this context. */
int rt_last_launch_count(rt_ctx *ctx);

/* Time of the last rt_sweep's traversal kernels only, in ms (cudaEvents on the sweep's stream);
   synchronises on those events.  When that sweep was replayed as one CUDA graph (rt_tune "graph"; see
   rt_last_sweep_was_graph) the interval is the whole sweep, normalisation kernel included.  Negative if unavailable,
   e.g. when the caller's stream was being captured (no timing events are recorded into a caller's graph). */
float rt_last_sweep_kernel_ms(rt_ctx *ctx);

/* 1 if the last rt_sweep of this context was replayed as one CUDA graph, 0 if its kernels were launched one by one. */
int rt_last_sweep_was_graph(rt_ctx *ctx);

/* Free everything the context owns.  Synchronises the device.  NULL is allowed. */
int rt_destroy(rt_ctx *ctx);

/* Static text for an RT_* code. */
const char *rt_strerror(int code);
/* Text of the last CUDA error seen by this thread in the library ("" if none). */
const char *rt_last_cuda_error(void);

#ifdef __cplusplus
}
#endif
#endif /* RT_H_ */
