// C ABI (include/rt.h) and host-side planner of the diffuse-radiation ray sweep.
// Host work here is O(N_d): direction records (PAPER.md:183 directions -> dominant axis, reflections,
// quantised slopes), batching of directions into launches, buffer management.  Everything that is
// O(N_m) or O(N_m N_d) runs in the kernels of rt_kernels.cu.
#include "../../include/rt.h"
#include "rt_internal.h"

#include <algorithm>
#include <cmath>
#include <cstring>
#include <map>
#include <new>
#include <tuple>
#include <string>
#include <vector>

using namespace rt;

static thread_local char g_cuda_err[256] = "";

static int cuda_fail(cudaError_t e)
{
    snprintf(g_cuda_err, sizeof(g_cuda_err), "%s: %s", cudaGetErrorName(e), cudaGetErrorString(e));
    return RT_ECUDA;
}
#define CK(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) return cuda_fail(e__); } while (0)
int rt::api_cuda_fail(cudaError_t e) { return cuda_fail(e); }

// Every entry point that takes a context makes the context's device current for the duration of the call (a
// process that drives several GPUs may have switched devices since rt_create) and restores the caller's.
struct DevGuard {
    int prev = -1;
    bool switched = false;
    explicit DevGuard(int dev)
    {
        if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) switched = (cudaSetDevice(dev) == cudaSuccess);
    }
    ~DevGuard() { if (switched) cudaSetDevice(prev); }
    DevGuard(const DevGuard &) = delete;
    DevGuard &operator=(const DevGuard &) = delete;
};

struct HostDir {
    int a, b, c;          // axes
    int refl[3];
    long long Mb, Mc;
    double L;
    int layout;           // 0 native, 1 transposed
    int Na, Nb, Nc;
    double work;          // 1 + mb + mc
    int parent;           // index of the direction in the caller's set
    int sub;              // alpha | beta << 8 | r << 16 (rt_internal.h sub_offset)
};

struct rt_ctx {
    int nx = 0, ny = 0, nz = 0, nbins = 1, ndirs = 0;
    int rays = 1;                    // r rays per cell width: every direction is r^2 unit sub-lattices ("virtual directions")
    int nv = 0;                      // ndirs * r^2: hd, d_dirs, d_prog and the batch lists are indexed by virtual direction
    long long ncell = 0;
    int pitch[2] = {0, 0};           // row pitch (cells) of the packed fields / accumulators of a layout: nx, ny padded to 32/64/128/256/512
    long long ncell_l[2] = {0, 0};   // cells per bin of a layout including the pad columns
    double cell_width = 1.0;
    unsigned flags = 0;
    int device = 0;
    int sm_count = 148;
    std::vector<HostDir> hd;
    std::vector<int> order[2];       // direction indices per layout, sorted by (dominant axis, march sense, work)
    // J sweep: directions that differ only by the sign of their b component are carried by one warp
    // ("mirror pairs", rt_kernels.cu); pairs[l] holds the member with a non-negative b component,
    // singles[l] everything that has no partner (zero b slope, or an unsymmetric user set)
    std::vector<int> pairs[2], singles[2];
    bool pair_enable = true;
    int handoff = 0;
    int slots_pair[2] = {0, 0}, slots_single[2] = {0, 0};
    int cap_pair[2] = {0, 0}, cap_single[2] = {0, 0};   // owned kernel: work items (CTAs per bin) of one full launch = one wave
    bool fast[2] = {false, false};   // owned kernel usable for the layout
    int pp[2] = {0, 0};              // packed field of the layout is pair-packed (rt_internal.h)
    int rows = 0;                    // rays rows per warp: 0 = by row width (1 up to 64 cells, 4 for 128, 2 for 256)
    int stages = 0;                  // depth of the owned kernel's TMA shared-memory ring: 0 = by row width (stages_for)
    int slots_req = 0;               // user override
    int slots[2] = {0, 0};           // allocated slots per layout
    bool fields_set = false;
    bool buffers_ready = false;
    // device
    DirDev *d_dirs = nullptr;
    double *d_L = nullptr;
    SlabProg *d_prog = nullptr;
    float2 *d_P[2] = {nullptr, nullptr};
    float *d_acc[2] = {nullptr, nullptr};
    float *d_accC[2] = {nullptr, nullptr};
    int *d_batch = nullptr;          // [2*ndirs]: order[0], order[1], then pairs[0], singles[0], pairs[1], singles[1]
    float *d_Ibc = nullptr;
    double *d_red = nullptr;         // [3] reduction scratch
    unsigned long long *d_u64 = nullptr;
    unsigned *d_cnt = nullptr;       // [ncell] scratch for rt_total_segments
    int np_max[2] = {0, 0}, nq_max[2] = {0, 0};
    int last_launches = 0;
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;
    bool ev_valid = false;
    bool last_graph = false;         // the last rt_sweep was a CUDA-graph replay: ev0 / ev1 then bracket the whole sweep
    // overlapped schedule (small meshes): every class of directions (layout, dominant axis, pairs / singles, march
    // sense along b) has its own slot range and runs on its own internal stream ("lane"), so that the classes of a
    // sweep that does not fill the machine run side by side instead of one short launch after the other
    struct ClassPlan { int l, pair, off, count, rev, Nc, tiles, slot_base, nslots, cap, lane, first; };
    int binpack = -1;                // rt_tune "binpack": -1 = automatic, 0 = bins are planes (one CTA per bin), 1 = three bins per row
    int nbp = 1;                     // bins packed per row of the packed fields and accumulators (1 or 3), fixed by ensure_buffers
    int wave_div = 0;                // overlapped schedule: work items per launch = one wave of resident CTAs / wave_div (0 = default)
    std::vector<ClassPlan> plan;
    int overlap = -1;                // rt_tune "overlap": -1 = automatic, 0 = off, 1 = on
    bool overlap_on = false;
    bool tiny = false;               // the whole sweep is at most two waves of resident CTAs: launch-latency bound, replayed as a CUDA graph
    int graph = -1;                  // rt_tune "graph": -1 = automatic (with the overlapped schedule), 0 = off, 1 = on
    static constexpr int kLanes = 8;
    cudaStream_t lane[kLanes] = {};
    cudaEvent_t ev_fork = nullptr, ev_join[kLanes] = {};
    cudaStream_t cap_stream = nullptr;   // origin stream of the graph captures (the caller's stream may be the legacy one)
    struct SweepGraph { float *J; unsigned what; int seen; cudaGraph_t graph; cudaGraphExec_t exec; };
    std::vector<SweepGraph> graphs;
    unsigned char *d_src = nullptr, *src_stage = nullptr;     // rt_point_sources: device tables {int src[n][3], float lum[n][nbins]} and pinned staging
    size_t src_cap = 0;
    int src_n = 0;
    bool src_valid = false, src_copy_pending = false;
    cudaEvent_t ev_src = nullptr;    // recorded after the copy into d_src: later calls on any stream wait on it before they read the tables
    std::map<cudaStream_t, cudaEvent_t> src_readers;   // per stream: recorded after its last kernel that reads d_src (a new copy waits on all)
    long long seg_total = -1;        // rt_total_segments: the geometry never changes, so the count is taken once
    unsigned long long *d_own = nullptr;   // [4] rt_debug_writer_counts: {max, sum} of acc, {max, sum} of accC
};

extern "C" const char *rt_strerror(int code)
{
    switch (code) {
    case RT_OK: return "ok";
    case RT_EINVAL: return "invalid argument";
    case RT_ENOMEM: return "out of memory";
    case RT_ECUDA: return "CUDA error";
    case RT_ESTATE: return "call order error";
    case RT_ELIMIT: return "size beyond the fixed capacity of a no-allocation entry point (RT_STATIC_MAX_*)";
    }
    return "unknown error";
}
extern "C" const char *rt_last_cuda_error(void) { return g_cuda_err; }

// HEALPix ring-scheme pixel centres; closed form of Gorski et al. (2005) as cited by PAPER.md:183.
extern "C" int rt_healpix_dirs(int nside, double *out)
{
    if (nside < 1 || nside > 8192 || !out) return RT_EINVAL;
    const double PI = 3.14159265358979323846;
    const double ns = (double)nside;
    int n = 0;
    for (int ring = 1; ring < 4 * nside; ++ring) {
        const bool north = ring < nside, south = ring > 3 * nside;
        const int ic = south ? 4 * nside - ring : ring;         // cap ring index counted from its pole
        const int count = (north || south) ? 4 * ic : 4 * nside;
        double z;
        if (north || south) z = 1.0 - (double)ic * ic / (3.0 * ns * ns);
        else z = 4.0 / 3.0 - 2.0 * ring / (3.0 * ns);
        const double rxy = std::sqrt((1.0 - z) * (1.0 + z));
        const double zz = south ? -z : z;
        for (int j = 1; j <= count; ++j) {
            double phi;
            if (north || south) phi = (j - 0.5) * PI / (2.0 * ic);
            else phi = (j - 0.5 * ((ring - nside + 1) % 2)) * PI / (2.0 * ns);
            out[3 * n + 0] = rxy * std::cos(phi);
            out[3 * n + 1] = rxy * std::sin(phi);
            out[3 * n + 2] = zz;
            ++n;
        }
    }
    return n;
}

static void free_device(rt_ctx *c)
{
    cudaFree(c->d_dirs); cudaFree(c->d_L); cudaFree(c->d_prog);
    for (int l = 0; l < 2; ++l) { cudaFree(c->d_P[l]); cudaFree(c->d_acc[l]); cudaFree(c->d_accC[l]); }
    cudaFree(c->d_batch); cudaFree(c->d_Ibc); cudaFree(c->d_red); cudaFree(c->d_u64); cudaFree(c->d_cnt); cudaFree(c->d_own);
    if (c->ev0) cudaEventDestroy(c->ev0);
    if (c->ev1) cudaEventDestroy(c->ev1);
    for (auto &g : c->graphs) { if (g.exec) cudaGraphExecDestroy(g.exec); if (g.graph) cudaGraphDestroy(g.graph); }
    c->graphs.clear();
    for (int i = 0; i < rt_ctx::kLanes; ++i) {
        if (c->lane[i]) cudaStreamDestroy(c->lane[i]);
        if (c->ev_join[i]) cudaEventDestroy(c->ev_join[i]);
    }
    if (c->ev_fork) cudaEventDestroy(c->ev_fork);
    cudaFree(c->d_src);
    if (c->src_stage) cudaFreeHost(c->src_stage);
    if (c->ev_src) cudaEventDestroy(c->ev_src);
    for (auto &kv : c->src_readers) cudaEventDestroy(kv.second);
    c->src_readers.clear();
    if (c->cap_stream) cudaStreamDestroy(c->cap_stream);
}

extern "C" int rt_create(rt_ctx **out, int nx, int ny, int nz, int nbins, const double *dirs, int ndirs,
                         int rays_per_cell, double cell_width, unsigned flags)
{
    if (!out) return RT_EINVAL;
    *out = nullptr;
    if (nx < 1 || ny < 1 || nz < 1 || nbins < 1 || nbins > 16 || !dirs || ndirs < 1) return RT_EINVAL;
    if (rays_per_cell < 1 || rays_per_cell > 16 || (rays_per_cell & (rays_per_cell - 1)) != 0) return RT_EINVAL;
    // per-cell segment counts (up to 3 per direction and sub-lattice) are tallied in fp32 accumulators: keep them exact
    if (3ll * ndirs * rays_per_cell * rays_per_cell >= (1ll << 24)) return RT_EINVAL;
    if (nx > (1 << 20) || ny > (1 << 20) || nz > (1 << 20)) return RT_EINVAL;
    if (!(cell_width > 0.0) || !std::isfinite(cell_width)) return RT_EINVAL;
    if (flags > 2u) return RT_EINVAL;
    if ((long long)nx * ny * nz >= (1ll << 31) || (long long)nx * ny * nz * nbins >= (1ll << 40)) return RT_EINVAL;
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess) return cuda_fail(e);
    if (ndev < 1) return cuda_fail(cudaErrorNoDevice);

    rt_ctx *c = new (std::nothrow) rt_ctx;
    if (!c) return RT_ENOMEM;
    c->nx = nx; c->ny = ny; c->nz = nz; c->nbins = nbins; c->ndirs = ndirs;
    c->rays = rays_per_cell;
    const int r2 = rays_per_cell * rays_per_cell, nv = ndirs * r2;
    c->nv = nv;
    c->ncell = (long long)nx * ny * nz; c->cell_width = cell_width; c->flags = flags;
    cudaGetDevice(&c->device);
    cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, c->device);
    const int dims[3] = {nx, ny, nz};
    // The owned kernel wants the memory-contiguous transverse extent to be 32/64/128/256/512: narrower or odd
    // rows are padded to the next such width (pad cells hold kappa = 0, S = 0: a ray crossing them keeps
    // its intensity and adds nothing, and a chain ray is replaced by the inflow where it wraps, after the pad).
    {
        const int NbL0[2] = {nx, ny};
        for (int l = 0; l < 2; ++l) {
            int p = NbL0[l];
            if (flags == RT_OWNED && p <= 512) { p = 32; while (p < NbL0[l]) p *= 2; }
            c->fast[l] = (flags == RT_OWNED) && NbL0[l] <= 512;
            c->pitch[l] = p;
            c->pp[l] = (c->fast[l] && p >= 64) ? 1 : 0;          // two columns per chunk
        }
        c->ncell_l[0] = (long long)c->pitch[0] * ny * nz;
        c->ncell_l[1] = (long long)c->pitch[1] * nz * nx;
        if (c->ncell_l[0] >= (1ll << 31) || c->ncell_l[1] >= (1ll << 31)) { delete c; return RT_EINVAL; }
    }

    // ---- direction records (reading O2): plain IEEE fp64 operations in a fixed order
    std::vector<DirDev> dd(nv);
    std::vector<double> Lv(nv);
    c->hd.resize(nv);
    long long prog_total = 0;
    for (int i = 0; i < nv; ++i) {
        const double *n = dirs + 3 * (i / r2);
        const double ab[3] = {std::fabs(n[0]), std::fabs(n[1]), std::fabs(n[2])};
        if (!(ab[0] > 0.0 || ab[1] > 0.0 || ab[2] > 0.0) || !std::isfinite(ab[0] + ab[1] + ab[2])) { delete c; return RT_EINVAL; }
        HostDir h;
        h.a = 0;
        if (ab[1] > ab[h.a]) h.a = 1;
        if (ab[2] > ab[h.a]) h.a = 2;
        h.b = (h.a == 0) ? 1 : 0;
        h.c = (h.a == 2) ? 1 : 2;
        for (int ax = 0; ax < 3; ++ax) h.refl[ax] = n[ax] < 0.0 ? 1 : 0;
        const double mb = ab[h.b] / ab[h.a], mc = ab[h.c] / ab[h.a];
        h.Mb = std::min<long long>(kOne, (long long)std::nearbyint(mb * (double)kOne));
        h.Mc = std::min<long long>(kOne, (long long)std::nearbyint(mc * (double)kOne));
        const double fb = (double)h.Mb / (double)kOne, fc = (double)h.Mc / (double)kOne;
        h.L = std::sqrt(1.0 + fb * fb + fc * fc);
        h.layout = (h.a == 0) ? 1 : 0;
        h.Na = dims[h.a]; h.Nb = dims[h.b]; h.Nc = dims[h.c];
        h.work = 1.0 + fb + fc;
        h.parent = i / r2;
        h.sub = rays_per_cell == 1 ? 0 : ((i % r2) % rays_per_cell) | (((i % r2) / rays_per_cell) << 8) | (rays_per_cell << 16);
        c->hd[i] = h;
        Lv[i] = h.L;

        // strides of the canonical axes in the layout this direction sweeps
        long long st[3];                       // element stride of x, y, z
        if (h.layout == 0) { st[0] = 1; st[1] = c->pitch[0]; st[2] = (long long)c->pitch[0] * ny; }          // [z][y][x]
        else               { st[1] = 1; st[2] = c->pitch[1]; st[0] = (long long)c->pitch[1] * nz; }          // [x][z][y]
        DirDev d;
        d.sk = st[h.a]; d.sl = st[h.c];
        d.base = 0;
        if (h.refl[h.a]) { d.base += (long long)(h.Na - 1) * d.sk; d.sk = -d.sk; }
        if (h.refl[h.c]) { d.base += (long long)(h.Nc - 1) * d.sl; d.sl = -d.sl; }
        d.sj = h.refl[h.b] ? -1 : 1;           // st[h.b] == 1 by construction of the layouts
        d.Na = h.Na; d.Nb = h.Nb; d.Nc = h.Nc;
        d.layout = h.layout | ((2 * h.a + h.refl[h.a]) << 8) | ((2 * h.b + h.refl[h.b]) << 12) | ((2 * h.c + h.refl[h.c]) << 16);
        d.prog_off = (int)prog_total;
        d.invL = (float)(1.0 / (h.L * cell_width * (double)r2));      // per cell and direction sum ds = r^2 L (pin P3)
        d.Mb = (int)h.Mb; d.Mc = (int)h.Mc; d.sub = h.sub;
        prog_total += h.Na;
        if (prog_total > 0x7fffffffll) { delete c; return RT_EINVAL; }
        dd[i] = d;
        c->order[h.layout].push_back(i);
        const int np = h.Nb + (int)((h.Na * h.Mb + kOne - 1) / kOne) + 1;
        const int nq = h.Nc + (int)((h.Na * h.Mc + kOne - 1) / kOne) + 1;
        c->np_max[h.layout] = std::max(c->np_max[h.layout], np);
        c->nq_max[h.layout] = std::max(c->nq_max[h.layout], nq);
    }
    // homogeneous batches: the directions of one launch share the dominant axis and the sense of the
    // march along it, so that concurrently resident CTAs read the same field slab at about the same
    // time (the second reader finds it in L2), and have similar work per slab
    auto by_class = [&](int x, int y) {
        if (c->hd[x].a != c->hd[y].a) return c->hd[x].a < c->hd[y].a;
        if (c->hd[x].refl[c->hd[x].a] != c->hd[y].refl[c->hd[y].a]) return c->hd[x].refl[c->hd[x].a] < c->hd[y].refl[c->hd[y].a];
        const int rx = c->hd[x].Mb == 0 ? 0 : c->hd[x].refl[c->hd[x].b], ry = c->hd[y].Mb == 0 ? 0 : c->hd[y].refl[c->hd[y].b];
        if (rx != ry) return rx < ry;
        return c->hd[x].work > c->hd[y].work;
    };
    for (int l = 0; l < 2; ++l) std::stable_sort(c->order[l].begin(), c->order[l].end(), by_class);
    // mirror pairs: same dominant axis, same reflections of a and c, same quantised slopes, opposite b
    {
        typedef std::tuple<int, int, int, long long, long long, int> Key;
        std::map<Key, std::vector<int>> pos, neg;
        for (int i = 0; i < nv; ++i) {
            const HostDir &h = c->hd[i];
            if (h.Mb == 0) continue;
            Key k(h.a, h.refl[h.a], h.refl[h.c], h.Mb, h.Mc, h.sub);     // same canonical sub-lattice offsets
            (h.refl[h.b] ? neg : pos)[k].push_back(i);
        }
        std::vector<char> paired(nv, 0);
        for (auto &kv : pos) {
            auto it = neg.find(kv.first);
            if (it == neg.end()) continue;
            const size_t n = std::min(kv.second.size(), it->second.size());
            for (size_t j = 0; j < n; ++j) {
                paired[kv.second[j]] = 1; paired[it->second[j]] = 2;
            }
        }
        for (int l = 0; l < 2; ++l)
            for (int i : c->order[l]) {
                if (paired[i] == 1) c->pairs[l].push_back(i);
                else if (paired[i] == 0) c->singles[l].push_back(i);
            }
    }
#define CKC(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) { int rc__ = (e__ == cudaErrorMemoryAllocation) ? RT_ENOMEM : cuda_fail(e__); free_device(c); delete c; return rc__; } } while (0)
    CKC(cudaMalloc(&c->d_dirs, sizeof(DirDev) * nv));
    CKC(cudaMalloc(&c->d_L, sizeof(double) * nv));
    CKC(cudaMalloc(&c->d_prog, sizeof(SlabProg) * prog_total));
    CKC(cudaMalloc(&c->d_batch, sizeof(int) * 2 * nv));
    CKC(cudaMalloc(&c->d_Ibc, sizeof(float) * 6 * nbins));
    CKC(cudaMalloc(&c->d_red, sizeof(double) * 3));
    CKC(cudaMalloc(&c->d_u64, sizeof(unsigned long long)));
    CKC(cudaMemset(c->d_Ibc, 0, sizeof(float) * 6 * nbins));
    CKC(cudaMemcpy(c->d_dirs, dd.data(), sizeof(DirDev) * nv, cudaMemcpyHostToDevice));
    CKC(cudaMemcpy(c->d_L, Lv.data(), sizeof(double) * nv, cudaMemcpyHostToDevice));
    {
        std::vector<int> batch;
        for (int l = 0; l < 2; ++l) batch.insert(batch.end(), c->order[l].begin(), c->order[l].end());
        for (int l = 0; l < 2; ++l) {
            batch.insert(batch.end(), c->pairs[l].begin(), c->pairs[l].end());
            batch.insert(batch.end(), c->singles[l].begin(), c->singles[l].end());
        }
        CKC(cudaMemcpy(c->d_batch, batch.data(), sizeof(int) * batch.size(), cudaMemcpyHostToDevice));
    }
    CKC(launch_build_programs(c->d_dirs, nv, std::max(nx, std::max(ny, nz)), c->d_prog, cell_width, c->d_L, 0));
    CKC(cudaEventCreate(&c->ev0));
    CKC(cudaEventCreate(&c->ev1));
    CKC(cudaDeviceSynchronize());
#undef CKC
    *out = c;
    return RT_OK;
}

extern "C" int rt_tune(rt_ctx *c, const char *key, int value)
{
    if (!c || !key) return RT_EINVAL;
    if (c->buffers_ready) return RT_ESTATE;
    if (!strcmp(key, "slots")) { if (value < 1 || value > 4096) return RT_EINVAL; c->slots_req = value; return RT_OK; }
    if (!strcmp(key, "stages")) { if (!(value >= 2 && value <= 4) || (c->handoff && value != 2)) return RT_EINVAL; c->stages = value; return RT_OK; }
    if (!strcmp(key, "handoff")) { if ((value != 0 && value != 1) || (value && c->stages != 2 && c->stages != 0)) return RT_EINVAL; c->handoff = value; if (value) c->stages = 2; return RT_OK; }
    if (!strcmp(key, "pair")) { if (value != 0 && value != 1) return RT_EINVAL; c->pair_enable = value != 0; return RT_OK; }
    if (!strcmp(key, "overlap")) { if (value < -1 || value > 1) return RT_EINVAL; c->overlap = value; return RT_OK; }
    if (!strcmp(key, "binpack")) { if (value < -1 || value > 1) return RT_EINVAL; c->binpack = value; return RT_OK; }
    if (!strcmp(key, "wave_div")) { if (value < 1 || value > 16) return RT_EINVAL; c->wave_div = value; return RT_OK; }
    if (!strcmp(key, "graph")) { if (value < -1 || value > 1) return RT_EINVAL; c->graph = value; return RT_OK; }
    if (!strcmp(key, "rows")) { if (!(value == 1 || value == 2 || value == 4)) return RT_EINVAL; c->rows = value; return RT_OK; }
    return RT_EINVAL;
}

// rows per warp actually used for a layout (must divide every Nc of the layout's directions)
static int rows_for(const rt_ctx *c, int layout)
{
    // by row width: short rows carry little work per warp and slab, so they want more warps (R = 1); 128-cell rows
    // fit four ray rows in the registers two 256-cell rows take
    int r = c->rows > 0 ? c->rows : (c->pitch[layout] == 128 ? 4 : (c->pitch[layout] <= 64 ? 1 : 2));
    if (c->pitch[layout] == 512) r = 1;                       // 512-cell rows: one ray row per warp fills the registers
    if (r == 4 && c->pitch[layout] > 128) r = 2;            // four rows per warp only fit the registers for rows of <= 128 cells
    if (c->nbp == 3) r = c->rows > 0 ? std::min(c->rows, 2) : (c->pitch[layout] == 128 ? kPackedRows128 : 1);   // three bins per row
    for (int i : c->order[layout])
        while (r > 1 && c->hd[i].Nc % r != 0) r >>= 1;
    return r;
}

// depth of the TMA ring used for a layout: rt_tune "stages", else by row width (a slab of a short row is little work
// per warp, so the copies of more slabs have to be in flight to cover their latency)
static int stages_for(const rt_ctx *c, int layout)
{
    if (c->stages > 0) return c->stages;
    return c->pitch[layout] <= 64 ? kShortRowStages : 2;
}

// Classes of a full J sweep in launch order (overlapped schedule).  The enumeration is the one run_traversal walks:
// per layout the mirror pairs, then the singles, cut where the dominant axis or the march sense along b changes.
// The classes of one (layout, dominant axis) share a lane (an internal stream) and a slot range: they run one after
// the other on that lane, so the slots of the first (largest) class serve the later ones too and the normalisation
// reads, and the seam clear writes, one range per lane instead of one per class.  false if some class cannot run on
// the owned kernel.
static bool build_overlap_plan(const rt_ctx *c, std::vector<rt_ctx::ClassPlan> &plan, int need[2], long long *items, bool share_lanes)
{
    plan.clear();
    need[0] = need[1] = 0;
    *items = 0;
    int lane_of[2][3], lane_base[2][3], lane_slots[2][3], nlanes = 0;
    for (int l = 0; l < 2; ++l) for (int a = 0; a < 3; ++a) lane_of[l][a] = -1;
    int off_all = 0, off_j = c->nv;
    for (int l = 0; l < 2; ++l) {
        const int nd = (int)c->order[l].size();
        const int my_all = off_all, my_j = off_j;
        off_all += nd;
        off_j += (int)(c->pairs[l].size() + c->singles[l].size());
        if (nd == 0) continue;
        if (!c->fast[l]) return false;
        const int rows = rows_for(c, l);
        const bool use_pairs = c->pair_enable && !c->pairs[l].empty();
        struct Pass { const std::vector<int> *list; int off; int S; int pair; };
        Pass passes[2];
        int npass = 0;
        if (use_pairs) {
            passes[npass++] = Pass{&c->pairs[l], my_j, c->slots_pair[l], 1};
            passes[npass++] = Pass{&c->singles[l], my_j + (int)c->pairs[l].size(), c->slots_single[l], 0};
        } else {
            passes[npass++] = Pass{&c->order[l], my_all, c->slots_single[l], 0};
        }
        for (int ps = 0; ps < npass; ++ps) {
            const std::vector<int> &list = *passes[ps].list;
            const int nl = (int)list.size();
            auto eff_rev = [&](int d) { return c->hd[d].Mb == 0 ? 0 : c->hd[d].refl[c->hd[d].b]; };
            int i = 0;
            while (i < nl) {
                const int a = c->hd[list[i]].a, rev = eff_rev(list[i]), Nc = c->hd[list[i]].Nc;
                if (!owned_supported(c->pitch[l], Nc, rows, c->nbp)) return false;
                int n = 0;
                while (i + n < nl && c->hd[list[i + n]].a == a && eff_rev(list[i + n]) == rev) ++n;
                rt_ctx::ClassPlan p;
                p.l = l; p.pair = passes[ps].pair; p.off = passes[ps].off + i; p.count = n; p.rev = rev; p.Nc = Nc;
                p.tiles = (Nc + kOwnedWarpsPerCta * rows - 1) / (kOwnedWarpsPerCta * rows);
                // launches of one wave / wave_div work items; a launch that starts anywhere touches at most
                // (cap - 1) / tiles + 2 entries, each of which needs a slot of its own
                const int wave = passes[ps].pair ? c->cap_pair[l] : c->cap_single[l];
                const int div = c->wave_div > 0 ? c->wave_div : kOverlapWaveDiv;
                p.cap = std::max(p.tiles, (wave > 0 ? wave : n * p.tiles) / div);
                int want = std::max(1, std::min(n, (p.cap - 1) / p.tiles + 2));
                if (want >= n) p.cap = n * p.tiles;              // every entry has its own slot: one launch
                // (a sweep of a wave or two is all launch latency: there every class gets a lane and slots of its own)
                p.first = !share_lanes || lane_of[l][a] < 0;
                if (p.first) {                                   // the lane's first class fixes its slot range
                    if (share_lanes && nlanes >= rt_ctx::kLanes) return false;
                    lane_of[l][a] = nlanes++ % rt_ctx::kLanes;
                    lane_base[l][a] = need[l];
                    lane_slots[l][a] = want;
                    need[l] += want;
                } else if (want > lane_slots[l][a]) {
                    // a later class lives in the slots the first one left: whole entries per launch, one slot to spare
                    want = lane_slots[l][a];
                    p.cap = std::max(1, want - 1) * p.tiles;
                }
                p.lane = lane_of[l][a];
                p.slot_base = lane_base[l][a];
                p.nslots = p.first ? want : lane_slots[l][a];
                *items += (long long)n * p.tiles * (c->nbins / c->nbp);
                plan.push_back(p);
                i += n;
            }
        }
    }
    return !plan.empty();
}

static int ensure_buffers(rt_ctx *c)
{
    if (c->buffers_ready) return RT_OK;
    // multi-bin packed rows: three bins of a cell row share the row (packed kernel), if every layout can run it
    c->nbp = 1;
    if (c->flags == RT_OWNED && c->nbins % 3 == 0 && !c->handoff && (c->stages == 0 || c->stages == 2) &&
        (c->binpack == 1 || (c->binpack == -1 && kBinpackDefault))) {
        bool ok = true;
        for (int l = 0; l < 2; ++l)
            if (!c->order[l].empty() && !(c->fast[l] && c->pitch[l] <= 128)) ok = false;
        // the packed kernel addresses a row's three bins with 32-bit element offsets scaled by 3 (rt_sweep.cuh):
        // larger layouts stay on bins-as-planes
        for (int l = 0; l < 2; ++l)
            if (3 * c->ncell_l[l] >= (1ll << 31)) ok = false;
        if (ok) c->nbp = 3;
    }
    // every layout that is swept by the owned kernel must have an instantiation for the rows / stages chosen with
    // rt_tune (e.g. a ring of 4 stages exists only for rows of <= 64 cells): refuse here, before anything is
    // allocated, so that the caller can still correct the knob
    if (c->flags == RT_OWNED)
        for (int l = 0; l < 2; ++l) {
            if (c->order[l].empty() || !c->fast[l]) continue;
            const int rows = rows_for(c, l), stages = stages_for(c, l);
            if (owned_ctas_per_sm(c->pitch[l], rows, stages, false, c->nbp) < 1 ||
                (c->pair_enable && owned_ctas_per_sm(c->pitch[l], rows, stages, true, c->nbp) < 1))
                return RT_EINVAL;
        }
    const size_t field_bytes_l[2] = {sizeof(float2) * (size_t)c->ncell_l[0] * c->nbins, sizeof(float2) * (size_t)c->ncell_l[1] * c->nbins};
    const size_t acc_bytes_l[2] = {sizeof(float) * (size_t)c->ncell_l[0] * c->nbins, sizeof(float) * (size_t)c->ncell_l[1] * c->nbins};
    size_t freeb = 0, totalb = 0;
    CK(cudaMemGetInfo(&freeb, &totalb));
    // slots: enough concurrent directions to fill the machine, bounded by memory (1/3 of free)
    for (int l = 0; l < 2; ++l) {
        const int nd = (int)c->order[l].size();
        int want = 0;
        if (nd > 0) {
            if (c->slots_req > 0) want = std::min(nd, c->slots_req);
            else {
                // one direction gives ceil(Nc/rows/4) CTAs per bin (owned kernel): fill the machine with
                // exactly one wave of resident CTAs, no partial second wave
                int Nc = c->hd[c->order[l][0]].Nc;
                for (int i : c->order[l]) Nc = std::min(Nc, c->hd[i].Nc);
                const int rows = rows_for(c, l);
                const int zgroups = c->nbins / c->nbp;               // grid.z of a J launch
                const int ctas_dir = ((Nc / rows + kOwnedWarpsPerCta - 1) / kOwnedWarpsPerCta) * zgroups;
                // A launch is one wave of resident CTAs, whole wave: `cap` work items (entry, row tile), not
                // rounded to whole entries; the entries of a launch cycle through cap / tiles + 2 slots.
                auto wave = [&](bool pair, int *cap) {
                    int per_sm = c->fast[l] ? owned_ctas_per_sm(c->pitch[l], rows, stages_for(c, l), pair, c->nbp) : 0;
                    if (per_sm < 1) per_sm = 4;
                    const int resident = per_sm * c->sm_count;
                    *cap = std::max(1, resident / std::max(1, zgroups));
                    // (a wave that is a whole number of entries needs no spare slots: launches then end on entry boundaries)
                    return std::max(1, std::min(nd, resident / std::max(1, ctas_dir) + ((resident % std::max(1, ctas_dir)) ? 2 : 0)));
                };
                c->slots_single[l] = wave(false, &c->cap_single[l]);
                c->slots_pair[l] = c->fast[l] ? wave(true, &c->cap_pair[l]) : 0;
                want = std::max(c->slots_single[l], c->slots_pair[l]);
                if (!c->fast[l]) want = std::min(nd, 16);
            }
            const size_t budget = freeb / 3;
            const size_t need_fixed = field_bytes_l[0] + field_bytes_l[1];
            size_t maxs = budget > need_fixed ? (budget - need_fixed) / (4 * acc_bytes_l[l]) : 1;
            if (maxs < 1) maxs = 1;
            want = (int)std::min<size_t>((size_t)want, maxs);
        }
        c->slots[l] = want;
        c->slots_single[l] = (c->slots_req > 0 || !c->fast[l]) ? want : std::min(want, c->slots_single[l]);
        c->slots_pair[l] = (c->slots_req > 0) ? want : std::min(want, c->slots_pair[l]);
    }
    // overlapped schedule: on by rt_tune, or by itself for meshes whose packed fields are L2-resident
    c->overlap_on = false;
    if (c->flags == RT_OWNED && c->overlap != 0 && c->slots_req == 0 && !c->handoff) {
        std::vector<rt_ctx::ClassPlan> plan;
        int need[2];
        long long items = 0;
        if (build_overlap_plan(c, plan, need, &items, false)) {
            long long capacity = 0;
            for (int l = 0; l < 2; ++l) capacity = std::max<long long>(capacity, (long long)std::max(c->cap_pair[l], c->cap_single[l]) * (c->nbins / c->nbp));
            const size_t budget = freeb / 3, need_fixed = field_bytes_l[0] + field_bytes_l[1];
            const size_t need_acc = 2 * (need[0] * acc_bytes_l[0] + need[1] * acc_bytes_l[1]);
            const bool fits = budget > need_fixed && need_acc <= budget - need_fixed;
            // by itself when the packed fields of both layouts stay in L2 next to the accumulator rows in flight (the
            // classes then need not march the same slabs to share them): measured C1 0.19 -> 0.07 ms, C2 0.74 -> 0.57 ms,
            // C3 7.31 -> 7.14 ms
            int l2_bytes = 0;
            cudaDeviceGetAttribute(&l2_bytes, cudaDevAttrL2CacheSize, c->device);
            const bool resident = need_fixed <= (size_t)l2_bytes / 2;
            c->tiny = items <= 2 * capacity;
            if (!c->tiny && !build_overlap_plan(c, plan, need, &items, true)) plan.clear();
            if ((c->overlap == 1 || (c->overlap == -1 && resident)) && fits && !plan.empty()) {
                c->plan.swap(plan);
                c->overlap_on = true;
                for (int l = 0; l < 2; ++l) c->slots[l] = std::max(c->slots[l], need[l]);
            }
        }
    }
    // on failure nothing stays allocated, so that a later call starts from scratch instead of leaking
    auto fail = [&](cudaError_t e) {
        for (int l = 0; l < 2; ++l) {
            cudaFree(c->d_P[l]); cudaFree(c->d_acc[l]); cudaFree(c->d_accC[l]);
            c->d_P[l] = nullptr; c->d_acc[l] = c->d_accC[l] = nullptr;
        }
        if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); return (int)RT_ENOMEM; }
        return cuda_fail(e);
    };
    for (int l = 0; l < 2; ++l) {
        {   // both packed copies are always kept (the pack kernel writes both in one pass)
            cudaError_t e = cudaMalloc(&c->d_P[l], field_bytes_l[l]);
            if (e == cudaSuccess) e = cudaMemset(c->d_P[l], 0, field_bytes_l[l]);      // pad cells stay zero
            if (e != cudaSuccess) return fail(e);
        }
        if (c->slots[l] > 0) {
            cudaError_t e = cudaMalloc(&c->d_acc[l], acc_bytes_l[l] * c->slots[l]);
            if (e == cudaSuccess) e = cudaMalloc(&c->d_accC[l], acc_bytes_l[l] * c->slots[l]);
            if (e != cudaSuccess) return fail(e);
        }
    }
    if (c->overlap_on) {
        cudaError_t e = cudaSuccess;
        for (int i = 0; i < rt_ctx::kLanes && e == cudaSuccess; ++i) {
            if (!c->lane[i]) e = cudaStreamCreateWithFlags(&c->lane[i], cudaStreamNonBlocking);
            if (e == cudaSuccess && !c->ev_join[i]) e = cudaEventCreateWithFlags(&c->ev_join[i], cudaEventDisableTiming);
        }
        if (e == cudaSuccess && !c->ev_fork) e = cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming);
        if (e == cudaSuccess && !c->cap_stream) e = cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking);
        if (e != cudaSuccess) return fail(e);
    }
    c->buffers_ready = true;
    return RT_OK;
}

extern "C" int rt_set_fields(rt_ctx *c, const float *kappa_dev, const float *S_dev, void *stream)
{
    if (!c || !kappa_dev || !S_dev) return RT_EINVAL;
    DevGuard dev_guard(c->device);
    int rc = ensure_buffers(c);
    if (rc != RT_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    CK(launch_pack_fields(kappa_dev, S_dev, c->d_P[0], c->d_P[1], c->pp[0], c->pp[1], c->nx, c->ny, c->nz, c->pitch[0], c->pitch[1], c->nbins, c->nbp, st));
    c->fields_set = true;
    return RT_OK;
}

extern "C" int rt_set_inflow(rt_ctx *c, const float *I_bc_host)
{
    if (!c || !I_bc_host) return RT_EINVAL;
    DevGuard dev_guard(c->device);
    std::vector<float> six(6 * (size_t)c->nbins);
    for (int b = 0; b < c->nbins; ++b) {
        if (!(I_bc_host[b] >= 0.0f) || !std::isfinite(I_bc_host[b])) return RT_EINVAL;
        for (int f = 0; f < 6; ++f) six[6 * (size_t)b + f] = I_bc_host[b];
    }
    CK(cudaDeviceSynchronize());        // sweeps in flight on any stream still read the old values
    CK(cudaMemcpy(c->d_Ibc, six.data(), sizeof(float) * six.size(), cudaMemcpyHostToDevice));
    return RT_OK;
}

extern "C" int rt_set_inflow_faces(rt_ctx *c, const float *I_face_host)
{
    if (!c || !I_face_host) return RT_EINVAL;
    DevGuard dev_guard(c->device);
    for (int i = 0; i < 6 * c->nbins; ++i) if (!(I_face_host[i] >= 0.0f) || !std::isfinite(I_face_host[i])) return RT_EINVAL;
    CK(cudaDeviceSynchronize());        // sweeps in flight on any stream still read the old values
    CK(cudaMemcpy(c->d_Ibc, I_face_host, sizeof(float) * 6 * c->nbins, cudaMemcpyHostToDevice));
    return RT_OK;
}

// Stream-ordered inflow update: the table (at most 16 bins x 6 faces) travels in the kernel's parameters, so there is no
// staging buffer to guard, nothing to synchronise and the caller's array is free when the call returns.
struct InflowTable { float v[6 * 16]; };
__global__ void k_set_inflow(float *__restrict__ Ibc, const InflowTable t, int n)
{
    const int i = threadIdx.x;
    if (i < n) Ibc[i] = t.v[i];
}

static int enqueue_inflow(rt_ctx *c, const InflowTable &t, cudaStream_t st)
{
    k_set_inflow<<<1, 6 * 16, 0, st>>>(c->d_Ibc, t, 6 * c->nbins);
    CK(cudaGetLastError());
    return RT_OK;
}

extern "C" int rt_set_inflow_async(rt_ctx *c, const float *I_bc_host, void *stream)
{
    if (!c || !I_bc_host) return RT_EINVAL;
    DevGuard dev_guard(c->device);
    InflowTable t = {};
    for (int b = 0; b < c->nbins; ++b) {
        if (!(I_bc_host[b] >= 0.0f) || !std::isfinite(I_bc_host[b])) return RT_EINVAL;
        for (int f = 0; f < 6; ++f) t.v[6 * b + f] = I_bc_host[b];
    }
    return enqueue_inflow(c, t, (cudaStream_t)stream);
}

extern "C" int rt_set_inflow_faces_async(rt_ctx *c, const float *I_face_host, void *stream)
{
    if (!c || !I_face_host) return RT_EINVAL;
    DevGuard dev_guard(c->device);
    InflowTable t = {};
    for (int i = 0; i < 6 * c->nbins; ++i) {
        if (!(I_face_host[i] >= 0.0f) || !std::isfinite(I_face_host[i])) return RT_EINVAL;
        t.v[i] = I_face_host[i];
    }
    return enqueue_inflow(c, t, (cudaStream_t)stream);
}

// Enqueue the traversal in `mode` of all directions (only_dir < 0) or of one direction (slot 0 of
// its layout).  The slot accumulators that will be used are zeroed first; used[l] receives the
// number of slots of layout l that hold results afterwards.
struct OwnerStats { unsigned long long launches = 0, partial = 0, expected = 0, entries = 0; };

static int run_traversal(rt_ctx *c, int mode, int only_dir, int nbins, cudaStream_t st, int *launches, int used[2],
                         OwnerStats *own = nullptr, bool record_events = true)
{
    const int r2 = c->rays * c->rays;
    used[0] = used[1] = 0;
    for (int l = 0; l < 2; ++l) {
        if (c->order[l].empty() || (only_dir >= 0 && c->hd[(size_t)only_dir * r2].layout != l)) continue;
        const int S = (only_dir >= 0) ? 1 : c->slots[l];
        const size_t acc_bytes = sizeof(float) * (size_t)c->ncell_l[l] * nbins;
        // the seam accumulator is written sparsely, so it is always cleared; the slot accumulators are cleared
        // below unless the first class of the layout initialises them itself (fresh entries)
        CK(cudaMemsetAsync(c->d_accC[l], 0, acc_bytes * S, st));
    }
    bool acc_ready[2] = {false, false};
    if (mode == MODE_J && record_events) CK(cudaEventRecord(c->ev0, st));
    int off_all = 0;                 // position of the layout's list in d_batch: order[] region ...
    int off_j = c->nv;            // ... and pairs[]/singles[] region
    for (int l = 0; l < 2; ++l) {
        const int nd = (int)c->order[l].size();
        const int my_all = off_all, my_j = off_j;
        off_all += nd;
        off_j += (int)(c->pairs[l].size() + c->singles[l].size());
        if (nd == 0) continue;
        if (only_dir >= 0 && c->hd[(size_t)only_dir * r2].layout != l) continue;
        SweepLaunch L;
        memset(&L, 0, sizeof(L));
        L.P = c->d_P[l]; L.acc = c->d_acc[l]; L.accC = c->d_accC[l];
        L.dirs = c->d_dirs; L.prog = c->d_prog; L.nbins = nbins; L.ncell = c->ncell_l[l]; L.Ibc = c->d_Ibc;
        L.rows = rows_for(c, l); L.mode = mode; L.stages = stages_for(c, l); L.handoff = c->handoff;
        L.Nb = c->pitch[l]; L.pp = c->pp[l];
        L.nbp = (nbins == c->nbins) ? c->nbp : 1;            // the counting modes run with one bin on plain rows
        const bool owned_l = c->fast[l];
        // the lists this traversal walks: (direction list, position in d_batch, slots per launch, paired)
        struct Pass { const std::vector<int> *list; int off; int S; int pair; };
        Pass passes[2];
        int npass = 0;
        const bool use_pairs = (mode == MODE_J || mode == MODE_OWNERS) && only_dir < 0 && c->pair_enable && owned_l &&
                               !c->pairs[l].empty();
        if (use_pairs) {
            passes[npass++] = Pass{&c->pairs[l], my_j, c->slots_pair[l], 1};
            passes[npass++] = Pass{&c->singles[l], my_j + (int)c->pairs[l].size(), c->slots_single[l], 0};
        } else {
            passes[npass++] = Pass{&c->order[l], my_all, (only_dir >= 0) ? 1 : c->slots_single[l], 0};
        }
        for (int ps = 0; ps < npass; ++ps) {
            const std::vector<int> &list = *passes[ps].list;
            const int nl = (int)list.size(), S = std::max(1, passes[ps].S);
            L.pair = passes[ps].pair;
            // batches never mix dominant axes (Nc differs between y- and z-dominant directions)
            int i = 0;
            while (i < nl) {
                // march sense along b: irrelevant for a zero b-slope (no ray ever changes column), so those
                // directions join forward batches whatever their sign
                auto eff_rev = [&](int d) { return c->hd[d].Mb == 0 ? 0 : c->hd[d].refl[c->hd[d].b]; };
                const int a = c->hd[list[i]].a;
                const int rev = eff_rev(list[i]);
                // owned kernel, full sweep: the batch is the whole class; it is cut into launches of work items below
                const bool whole = owned_l && only_dir < 0 && owned_supported(L.Nb, c->hd[list[i]].Nc, L.rows, L.nbp);
                int n = 0;
                while (i + n < nl && (whole || n < S) && c->hd[list[i + n]].a == a && eff_rev(list[i + n]) == rev) ++n;
                int first = i, count = n;
                if (only_dir >= 0) {
                    if (c->hd[list[i]].parent != only_dir) { i += 1; continue; }      // all r^2 sub-lattices, one by one
                    count = 1;
                }
                used[l] = std::max(used[l], whole ? std::min(count, std::max(1, c->slots[l])) : count);
                if (!acc_ready[l]) {
                    // first launches of the layout in this traversal
                    const int S0 = (only_dir >= 0) ? 1 : c->slots[l];
                    const bool self_init = whole && mode == MODE_J && !c->handoff && count >= std::max(1, c->slots[l]);
                    if (!self_init) CK(cudaMemsetAsync(c->d_acc[l], 0, sizeof(float) * (size_t)c->ncell_l[l] * nbins * S0, st));
                    L.fresh_below = self_init ? std::max(1, c->slots[l]) : 0;
                    acc_ready[l] = true;
                } else L.fresh_below = 0;
                L.batch = c->d_batch + passes[ps].off + first;
                L.nslots = count;
                L.rev = rev;
                L.Nc = c->hd[list[first]].Nc;
                if (owned_l && owned_supported(L.Nb, L.Nc, L.rows, L.nbp)) {
                    const int tiles = (L.Nc + kOwnedWarpsPerCta * L.rows - 1) / (kOwnedWarpsPerCta * L.rows);
                    L.tiles = tiles;
                    if (only_dir >= 0) {
                        L.nslots = 1; L.item0 = 0; L.nitems = tiles;
                        CK(launch_sweep_owned(L, st));
                        ++*launches;
                    } else {
                        // work items (entry, row tile) of the class, one resident wave per launch; a launch may
                        // start and end inside an entry, and touches at most nslots entries
                        const int nsl = std::max(1, c->slots[l]);
                        int cap = L.pair ? c->cap_pair[l] : c->cap_single[l];
                        if (c->slots_req > 0 || cap < 1) cap = nsl * tiles;            // whole entries per launch
                        else if (cap % tiles == 0) cap = std::max(tiles, std::min(cap, nsl * tiles));
                        else cap = std::max(tiles, std::min(cap, (nsl - 1) * tiles));
                        if (nsl == 1) cap = tiles;
                        L.nslots = nsl;
                        const long long total = (long long)count * tiles;
                        for (long long item0 = 0; item0 < total; item0 += cap) {
                            L.item0 = (int)item0;
                            L.nitems = (int)std::min<long long>(cap, total - item0);
                            const size_t nacc = (size_t)c->ncell_l[l] * nbins * nsl;
                            if (mode == MODE_OWNERS) {       // writer counts of this launch alone
                                CK(cudaMemsetAsync(c->d_acc[l], 0, sizeof(float) * nacc, st));
                                CK(cudaMemsetAsync(c->d_accC[l], 0, sizeof(float) * nacc, st));
                            }
                            CK(launch_sweep_owned(L, st));
                            ++*launches;
                            if (mode == MODE_OWNERS) {
                                CK(launch_owner_reduce(c->d_own, c->d_acc[l], (long long)nacc, st));
                                CK(launch_owner_reduce(c->d_own + 2, c->d_accC[l], (long long)nacc, st));
                                own->launches += 1;
                                if (L.item0 % tiles != 0 || (L.item0 + L.nitems) % tiles != 0) own->partial += 1;
                            }
                        }
                        if (mode == MODE_OWNERS) {
                            own->entries += (unsigned long long)count;
                            own->expected += (unsigned long long)count * (unsigned long long)c->ncell_l[l] * (unsigned long long)nbins;
                        }
                        used[l] = std::max(used[l], std::min(nsl, count));
                    }
                } else if (mode == MODE_OWNERS) {
                    return RT_EINVAL;                 // the writer-count check is for the owned kernel's ownership scheme
                } else if (c->flags == RT_ATOMIC_ABLATION) {
                    L.variant = 1;
                    CK(launch_sweep_generic(L, c->np_max[l], c->nq_max[l], st));
                    ++*launches;
                } else {
                    L.variant = 0;
                    for (int g = 0; g < 4; ++g) {
                        L.group = g;
                        CK(launch_sweep_generic(L, c->np_max[l], c->nq_max[l], st));
                        ++*launches;
                    }
                }
                i += count;
            }
        }
    }
    if (mode == MODE_J && record_events) { CK(cudaEventRecord(c->ev1, st)); c->ev_valid = true; }
    return RT_OK;
}

// Overlapped J sweep (ensure_buffers decided c->overlap_on): the lanes of the plan (one per layout and dominant axis)
// run side by side on the context's internal streams, forked from and joined back into `st` with events; the classes
// of a lane run one after the other in its slot range.  The first class of a lane starts the slots from zero
// ("fresh" entries), so no slot accumulator is cleared; the sparsely written seam accumulators are.
static int run_overlapped(rt_ctx *c, cudaStream_t st, int *launches, int used[2], bool record_events,
                          OwnerStats *own = nullptr)
{
    const int nbins = c->nbins;
    const int mode = own ? MODE_OWNERS : MODE_J;           // writer-count check: same launches, one after the other on st
    for (int l = 0; l < 2; ++l) {
        used[l] = 0;
        for (const auto &p : c->plan) if (p.l == l) used[l] = std::max(used[l], p.slot_base + p.nslots);
        if (used[l] > 0) CK(cudaMemsetAsync(c->d_accC[l], 0, sizeof(float) * (size_t)c->ncell_l[l] * nbins * used[l], st));
    }
    if (record_events) CK(cudaEventRecord(c->ev0, st));
    if (!own) CK(cudaEventRecord(c->ev_fork, st));
    bool lane_used[rt_ctx::kLanes] = {};
    for (const auto &p : c->plan) {
        const int ln = p.lane;
        cudaStream_t ls = own ? st : c->lane[ln];
        if (!own && !lane_used[ln]) { CK(cudaStreamWaitEvent(ls, c->ev_fork, 0)); lane_used[ln] = true; }
        const int l = p.l;
        SweepLaunch L;
        memset(&L, 0, sizeof(L));
        const size_t slot_stride = (size_t)c->ncell_l[l] * nbins;
        L.P = c->d_P[l]; L.acc = c->d_acc[l] + slot_stride * p.slot_base; L.accC = c->d_accC[l] + slot_stride * p.slot_base;
        L.dirs = c->d_dirs; L.prog = c->d_prog; L.nbins = nbins; L.ncell = c->ncell_l[l]; L.Ibc = c->d_Ibc;
        L.rows = rows_for(c, l); L.mode = mode; L.stages = stages_for(c, l); L.handoff = 0;
        L.Nb = c->pitch[l]; L.pp = c->pp[l]; L.nbp = c->nbp; L.pair = p.pair; L.rev = p.rev; L.Nc = p.Nc; L.tiles = p.tiles;
        L.batch = c->d_batch + p.off;
        L.nslots = p.nslots;
        // the first class of a lane starts its slots from zero ("fresh" entries: it has at least nslots entries, and an
        // entry writes every cell of its slot); the later classes of the lane add to what it left
        L.fresh_below = p.first ? p.nslots : 0;
        const int cap = p.cap;
        const long long total = (long long)p.count * p.tiles;
        const size_t nacc = slot_stride * p.nslots;
        for (long long item0 = 0; item0 < total; item0 += cap) {
            L.item0 = (int)item0;
            L.nitems = (int)std::min<long long>(cap, total - item0);
            if (own) {                                       // writer counts of this launch alone
                CK(cudaMemsetAsync(L.acc, 0, sizeof(float) * nacc, ls));
                CK(cudaMemsetAsync(L.accC, 0, sizeof(float) * nacc, ls));
            }
            CK(launch_sweep_owned(L, ls));
            ++*launches;
            if (own) {
                CK(launch_owner_reduce(c->d_own, L.acc, (long long)nacc, ls));
                CK(launch_owner_reduce(c->d_own + 2, L.accC, (long long)nacc, ls));
                own->launches += 1;
                if (L.item0 % p.tiles != 0 || (L.item0 + L.nitems) % p.tiles != 0) own->partial += 1;
            }
        }
        if (own) {
            own->entries += (unsigned long long)p.count;
            own->expected += (unsigned long long)p.count * (unsigned long long)slot_stride;
        }
    }
    for (int ln = 0; ln < rt_ctx::kLanes; ++ln)
        if (lane_used[ln]) {
            CK(cudaEventRecord(c->ev_join[ln], c->lane[ln]));
            CK(cudaStreamWaitEvent(st, c->ev_join[ln], 0));
        }
    if (record_events) { CK(cudaEventRecord(c->ev1, st)); c->ev_valid = true; }
    return RT_OK;
}

// traversal + normalisation of one rt_sweep, enqueued on st
static int enqueue_sweep(rt_ctx *c, float *J_dev, unsigned what, cudaStream_t st, bool record_events)
{
    int launches = 0;
    int used[2];
    int rc = c->overlap_on ? run_overlapped(c, st, &launches, used, record_events)
                           : run_traversal(c, MODE_J, -1, c->nbins, st, &launches, used, nullptr, record_events);
    if (rc != RT_OK) return rc;
    CK(launch_normalise(J_dev, c->d_P[0], c->pp[0], c->d_acc[0], c->d_accC[0], used[0], c->d_acc[1], c->d_accC[1], used[1],
                        c->nx, c->ny, c->nz, c->pitch[0], c->pitch[1], c->nbins, c->nbp, what == RT_SUM_IN ? 1.0f : (float)(1.0 / (double)c->ndirs),
                        what == RT_J_TOTAL ? 1 : 0, st));
    c->last_launches = launches + 1;
    return RT_OK;
}

extern "C" int rt_sweep(rt_ctx *c, float *J_dev, unsigned what, void *stream)
{
    if (!c || !J_dev || what > 2u) return RT_EINVAL;
    DevGuard dev_guard(c->device);
    if (!c->fields_set) return RT_ESTATE;
    cudaStream_t st = (cudaStream_t)stream;
    // A sweep of a few short launches is bound by launch latency: from its second use on, a (J buffer, what)
    // combination is replayed as one CUDA graph (captured on an internal stream, launched into the caller's).
    const bool want_graph = c->graph == 1 || (c->graph == -1 && c->overlap_on && c->tiny);
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    if (st != nullptr && st != cudaStreamLegacy && st != cudaStreamPerThread) CK(cudaStreamIsCapturing(st, &cap));
    c->last_graph = false;
    if (cap != cudaStreamCaptureStatusNone) {
        // the caller is capturing this stream: timing events recorded now would become nodes of the caller's graph and
        // could never be read back, so none are recorded and rt_last_sweep_kernel_ms reports "unavailable"
        c->ev_valid = false;
        return enqueue_sweep(c, J_dev, what, st, false);
    }
    if (want_graph) {
        if (!c->cap_stream) CK(cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking));
        rt_ctx::SweepGraph *g = nullptr;
        for (auto &e : c->graphs) if (e.J == J_dev && e.what == what) g = &e;
        if (!g) {
            if (c->graphs.size() >= 8) {                          // forget the oldest combination
                if (c->graphs[0].exec) cudaGraphExecDestroy(c->graphs[0].exec);
                if (c->graphs[0].graph) cudaGraphDestroy(c->graphs[0].graph);
                c->graphs.erase(c->graphs.begin());
            }
            c->graphs.push_back(rt_ctx::SweepGraph{J_dev, what, 0, nullptr, nullptr});
            g = &c->graphs.back();
        }
        if (g->seen >= 1 && !g->exec) {
            CK(cudaStreamBeginCapture(c->cap_stream, cudaStreamCaptureModeThreadLocal));
            int rc = enqueue_sweep(c, J_dev, what, c->cap_stream, false);
            cudaGraph_t graph = nullptr;
            cudaError_t e = cudaStreamEndCapture(c->cap_stream, &graph);
            if (rc != RT_OK) { if (graph) cudaGraphDestroy(graph); return rc; }
            if (e != cudaSuccess) return cuda_fail(e);
            e = cudaGraphInstantiate(&g->exec, graph, 0);
            if (e != cudaSuccess) { cudaGraphDestroy(graph); g->exec = nullptr; return cuda_fail(e); }
            g->graph = graph;
        }
        g->seen += 1;
        if (g->exec) {
            CK(cudaEventRecord(c->ev0, st));
            CK(cudaGraphLaunch(g->exec, st));
            CK(cudaEventRecord(c->ev1, st));
            c->ev_valid = true;                                   // here the events bracket the whole sweep, normalisation included
            c->last_graph = true;
            return RT_OK;
        }
    }
    return enqueue_sweep(c, J_dev, what, st, true);
}

extern "C" int rt_combine(rt_ctx *c, const float *sum_dev, long long ndirs_total, unsigned what, float *J_dev, void *stream)
{
    if (!c || !sum_dev || !J_dev || ndirs_total < 1 || what > 1u) return RT_EINVAL;
    DevGuard dev_guard(c->device);
    if (!c->fields_set) return RT_ESTATE;
    CK(launch_combine(J_dev, sum_dev, c->d_P[0], c->pp[0], c->nx, c->ny, c->nz, c->pitch[0], c->nbins, c->nbp, (float)(1.0 / (double)ndirs_total),
                      what == RT_J_TOTAL ? 1 : 0, (cudaStream_t)stream));
    return RT_OK;
}

extern "C" int rt_sweep_rates(rt_ctx *c, float *Gamma_dev, float *Heat_dev, const double *wG, const double *lG,
                              const double *wH, const double *lH, void *stream)
{
    if (!c || !Gamma_dev || !Heat_dev || !wG || !lG || !wH || !lH) return RT_EINVAL;
    DevGuard dev_guard(c->device);
    if (!c->fields_set) return RT_ESTATE;
    std::vector<float> w4(4 * (size_t)c->nbins);
    const double *src[4] = {wG, lG, wH, lH};
    for (int k = 0; k < 4; ++k)
        for (int b = 0; b < c->nbins; ++b) {
            if (!std::isfinite(src[k][b])) return RT_EINVAL;
            w4[(size_t)k * c->nbins + b] = (float)src[k][b];
        }
    cudaStream_t st = (cudaStream_t)stream;
    int launches = 0;
    int used[2];
    int rc = c->overlap_on ? run_overlapped(c, st, &launches, used, true)
                           : run_traversal(c, MODE_J, -1, c->nbins, st, &launches, used);
    if (rc != RT_OK) return rc;
    CK(launch_rates(Gamma_dev, Heat_dev, c->d_P[0], c->pp[0], c->d_acc[0], c->d_accC[0], used[0], c->d_acc[1], c->d_accC[1],
                    used[1], c->nx, c->ny, c->nz, c->pitch[0], c->pitch[1], c->nbins, c->nbp, (float)(1.0 / (double)c->ndirs), w4.data(), st));
    c->last_launches = launches + 1;
    return RT_OK;
}

// Source tables of rt_point_sources: persistent device copies, refilled only when the caller's tables change, through a
// context-owned pinned staging buffer, so that the call only enqueues (no allocation, no synchronisation).
static int upload_sources(rt_ctx *c, const int *src_fix_host, const float *lum, int nsrc, cudaStream_t st)
{
    const size_t nsrc3 = 3 * (size_t)nsrc, nlum = (size_t)nsrc * c->nbins;
    const size_t bytes = sizeof(int) * nsrc3 + sizeof(float) * nlum;
    if (c->src_valid && c->src_n == nsrc && !memcmp(c->src_stage, src_fix_host, sizeof(int) * nsrc3) &&
        !memcmp(c->src_stage + sizeof(int) * nsrc3, lum, sizeof(float) * nlum))
    {                                                            // same sources as last time: the device tables stand, but the
        if (c->ev_src) CK(cudaStreamWaitEvent(st, c->ev_src, 0));  // copy that filled them may be in flight on another stream
        return RT_OK;
    }
    if (c->src_copy_pending) { CK(cudaEventSynchronize(c->ev_src)); c->src_copy_pending = false; }   // staging buffer still being read
    if (bytes > c->src_cap) {
        CK(cudaDeviceSynchronize());                             // kernels in flight may still read the old tables
        cudaFree(c->d_src); c->d_src = nullptr;
        if (c->src_stage) cudaFreeHost(c->src_stage);
        c->src_stage = nullptr; c->src_cap = 0; c->src_valid = false;
        const size_t cap = std::max<size_t>(2 * bytes, 4096);
        cudaError_t e = cudaMalloc(&c->d_src, cap);
        if (e == cudaSuccess) e = cudaMallocHost(&c->src_stage, cap);
        if (e != cudaSuccess) { cudaFree(c->d_src); c->d_src = nullptr; return e == cudaErrorMemoryAllocation ? RT_ENOMEM : cuda_fail(e); }
        c->src_cap = cap;
        if (!c->ev_src) CK(cudaEventCreateWithFlags(&c->ev_src, cudaEventDisableTiming));
    }
    // kernels of earlier calls, on whatever stream they ran, may still be reading the tables this copy overwrites
    for (auto &kv : c->src_readers)
        if (kv.first != st) CK(cudaStreamWaitEvent(st, kv.second, 0));
    memcpy(c->src_stage, src_fix_host, sizeof(int) * nsrc3);
    memcpy(c->src_stage + sizeof(int) * nsrc3, lum, sizeof(float) * nlum);
    CK(cudaMemcpyAsync(c->d_src, c->src_stage, bytes, cudaMemcpyHostToDevice, st));
    CK(cudaEventRecord(c->ev_src, st));
    c->src_copy_pending = true;
    c->src_n = nsrc; c->src_valid = true;
    return RT_OK;
}

// Remember that a kernel reading d_src has been enqueued on `st` (one event per stream, re-recorded by every call).
static int note_source_reader(rt_ctx *c, cudaStream_t st)
{
    auto it = c->src_readers.find(st);
    if (it == c->src_readers.end()) {
        if (c->src_readers.size() >= 64) {                       // a caller cycling through many streams: wait for all readers once, start over
            for (auto &kv : c->src_readers) { cudaEventSynchronize(kv.second); cudaEventDestroy(kv.second); }
            c->src_readers.clear();
        }
        cudaEvent_t ev = nullptr;
        CK(cudaEventCreateWithFlags(&ev, cudaEventDisableTiming));
        it = c->src_readers.emplace(st, ev).first;
    }
    CK(cudaEventRecord(it->second, st));
    return RT_OK;
}

extern "C" int rt_point_sources(rt_ctx *c, const int *src_fix_host, const double *lum_host, int nsrc, float *Q_dev,
                                int diag_src, int diag_bin, float *tau_dev, unsigned long long *steps_host, void *stream)
{
    if (!c || !src_fix_host || !lum_host || nsrc < 1 || nsrc > (1 << 20) || !Q_dev) return RT_EINVAL;
    DevGuard dev_guard(c->device);
    if (c->nx > 1024 || c->ny > 1024 || c->nz > 1024) return RT_EINVAL;       // crossing parameters below 2^54
    if (tau_dev && (diag_src < 0 || diag_src >= nsrc || diag_bin < 0 || diag_bin >= c->nbins)) return RT_EINVAL;
    if (!c->fields_set) return RT_ESTATE;
    const int dims[3] = {c->nx, c->ny, c->nz};
    std::vector<float> lum((size_t)nsrc * c->nbins);
    for (int a = 0; a < nsrc; ++a) {
        for (int i = 0; i < 3; ++i)
            if (src_fix_host[3 * a + i] < 0 || src_fix_host[3 * a + i] > dims[i] * 256) return RT_EINVAL;
        for (int b = 0; b < c->nbins; ++b) {
            const double v = lum_host[(size_t)a * c->nbins + b];
            if (!(v >= 0.0) || !std::isfinite(v)) return RT_EINVAL;
            lum[(size_t)a * c->nbins + b] = (float)v;
        }
    }
    cudaStream_t st = (cudaStream_t)stream;
    int rc = upload_sources(c, src_fix_host, lum.data(), nsrc, st);
    if (rc != RT_OK) return rc;
    const int *d_src = reinterpret_cast<const int *>(c->d_src);
    const float *d_lum = reinterpret_cast<const float *>(c->d_src + sizeof(int) * 3 * (size_t)nsrc);
    if (steps_host) CK(cudaMemsetAsync(c->d_u64, 0, sizeof(unsigned long long), st));
    CK(launch_point_sources(Q_dev, tau_dev, c->d_P[0], c->pp[0], c->nx, c->ny, c->nz, c->pitch[0], d_src, d_lum, nsrc,
                            c->nbins, c->nbp, (float)c->cell_width, diag_src, diag_bin, steps_host ? c->d_u64 : nullptr, st));
    rc = note_source_reader(c, st);
    if (rc != RT_OK) return rc;
    c->last_launches = 1;
    if (steps_host) {                                            // the one synchronising variant: the count comes back to the host
        CK(cudaMemcpyAsync(steps_host, c->d_u64, sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
    }
    return RT_OK;
}

extern "C" int rt_point_source_rates(rt_ctx *c, const float *Q_dev, const float *kappa_sp_dev, const float *n_sp_dev, int nspecies,
                                     const double *hnu_host, const double *hnu_thr_host, float *Gamma_dev, float *Heat_dev, void *stream)
{
    if (!c || !Q_dev || !kappa_sp_dev || !n_sp_dev || !hnu_host || !hnu_thr_host || !Gamma_dev || !Heat_dev) return RT_EINVAL;
    if (nspecies < 1 || nspecies > kMaxSpecies) return RT_EINVAL;
    DevGuard dev_guard(c->device);
    if (!c->fields_set) return RT_ESTATE;
    SpeciesWeights W;
    memset(&W, 0, sizeof(W));
    for (int b = 0; b < c->nbins; ++b)
        if (!(hnu_host[b] > 0.0) || !std::isfinite(hnu_host[b])) return RT_EINVAL;
    for (int s = 0; s < nspecies; ++s) {
        if (!(hnu_thr_host[s] >= 0.0) || !std::isfinite(hnu_thr_host[s])) return RT_EINVAL;
        for (int b = 0; b < c->nbins; ++b)
            if (hnu_host[b] >= hnu_thr_host[s]) {              // the integrals of eqs. A5-A6 start at the threshold
                W.wG[s][b] = (float)(1.0 / hnu_host[b]);
                W.wH[s][b] = (float)((hnu_host[b] - hnu_thr_host[s]) / hnu_host[b]);
            }
    }
    CK(launch_point_source_rates(Gamma_dev, Heat_dev, Q_dev, kappa_sp_dev, n_sp_dev, c->d_P[0], c->pp[0], c->nx, c->ny, c->nz,
                                 c->pitch[0], c->nbins, c->nbp, nspecies, W, c->sm_count, (cudaStream_t)stream));
    c->last_launches = 1;
    return RT_OK;
}

extern "C" int rt_segment_counts(rt_ctx *c, int dir_index, unsigned int *counts_dev, void *stream)
{
    if (!c || !counts_dev || dir_index < -1 || dir_index >= c->ndirs) return RT_EINVAL;
    DevGuard dev_guard(c->device);
    int rc = ensure_buffers(c);
    if (rc != RT_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    int launches = 0;
    int used[2];
    rc = run_traversal(c, MODE_COUNT, dir_index, 1, st, &launches, used);
    if (rc != RT_OK) return rc;
    CK(launch_counts_finalise(counts_dev, c->d_acc[0], c->d_accC[0], used[0], c->d_acc[1], c->d_accC[1], used[1],
                              c->nx, c->ny, c->nz, c->pitch[0], c->pitch[1], st));
    return RT_OK;
}

extern "C" int rt_debug_writer_counts(rt_ctx *c, unsigned long long *out_host, void *stream)
{
    if (!c || !out_host) return RT_EINVAL;
    if (c->flags != RT_OWNED) return RT_EINVAL;
    DevGuard dev_guard(c->device);
    int rc = ensure_buffers(c);
    if (rc != RT_OK) return rc;
    for (int l = 0; l < 2; ++l)           // every layout must run on the owned kernel (rows <= 512 cells)
        if (!c->order[l].empty() && !c->fast[l]) return RT_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    if (!c->d_own) {
        cudaError_t e = cudaMalloc(&c->d_own, sizeof(unsigned long long) * 4);
        if (e != cudaSuccess) return e == cudaErrorMemoryAllocation ? RT_ENOMEM : cuda_fail(e);
    }
    CK(cudaMemsetAsync(c->d_own, 0, sizeof(unsigned long long) * 4, st));
    OwnerStats own;
    int launches = 0, used[2];
    rc = c->overlap_on ? run_overlapped(c, st, &launches, used, false, &own)
                       : run_traversal(c, MODE_OWNERS, -1, c->nbins, st, &launches, used, &own);
    if (rc != RT_OK) return rc;
    unsigned long long dev[4];
    CK(cudaMemcpyAsync(dev, c->d_own, sizeof(dev), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    out_host[0] = dev[0]; out_host[1] = dev[1]; out_host[2] = dev[2]; out_host[3] = dev[3];
    out_host[4] = own.launches; out_host[5] = own.partial; out_host[6] = own.expected; out_host[7] = own.entries;
    return RT_OK;
}

extern "C" int rt_total_segments(rt_ctx *c, unsigned long long *n_host, void *stream)
{
    if (!c || !n_host) return RT_EINVAL;
    if (c->seg_total >= 0) { *n_host = (unsigned long long)c->seg_total; return RT_OK; }
    DevGuard dev_guard(c->device);
    cudaStream_t st = (cudaStream_t)stream;
    if (!c->d_cnt) {
        cudaError_t e = cudaMalloc(&c->d_cnt, sizeof(unsigned) * (size_t)c->ncell);
        if (e != cudaSuccess) return e == cudaErrorMemoryAllocation ? RT_ENOMEM : cuda_fail(e);
    }
    int rc = rt_segment_counts(c, -1, c->d_cnt, stream);
    if (rc != RT_OK) return rc;
    CK(cudaMemsetAsync(c->d_u64, 0, sizeof(unsigned long long), st));
    CK(launch_sum_u32(c->d_u64, c->d_cnt, c->ncell, st));
    CK(cudaMemcpyAsync(n_host, c->d_u64, sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    c->seg_total = (long long)*n_host;
    cudaFree(c->d_cnt);                  // the scratch is not needed again
    c->d_cnt = nullptr;
    return RT_OK;
}

extern "C" int rt_sum_ds(rt_ctx *c, double *sum_host, double *min_host, double *max_host, void *stream)
{
    if (!c || !sum_host) return RT_EINVAL;
    DevGuard dev_guard(c->device);
    int rc = ensure_buffers(c);
    if (rc != RT_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    std::vector<double> res(3 * (size_t)c->ndirs);
    double *d_all = nullptr;
    cudaError_t e = cudaMalloc(&d_all, sizeof(double) * 3 * (size_t)c->ndirs);
    if (e != cudaSuccess) return e == cudaErrorMemoryAllocation ? RT_ENOMEM : cuda_fail(e);
    {
        std::vector<double> init(3 * (size_t)c->ndirs);
        for (int i = 0; i < c->ndirs; ++i) { init[3 * i] = 0.0; init[3 * i + 1] = 1.0e300; init[3 * i + 2] = 0.0; }
        e = cudaMemcpyAsync(d_all, init.data(), sizeof(double) * init.size(), cudaMemcpyHostToDevice, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) { cudaFree(d_all); return cuda_fail(e); }
    }
    for (int i = 0; i < c->ndirs; ++i) {
        int launches = 0, used[2];
        rc = run_traversal(c, MODE_DS, i, 1, st, &launches, used);
        if (rc != RT_OK) { cudaFree(d_all); return rc; }
        const int l = c->hd[(size_t)i * c->rays * c->rays].layout;
        e = launch_ds_reduce(d_all + 3 * i, c->d_acc[l], c->d_accC[l], c->ncell_l[l], c->pitch[l], l == 0 ? c->nx : c->ny, st);
        if (e != cudaSuccess) { cudaFree(d_all); return cuda_fail(e); }
    }
    e = cudaMemcpyAsync(res.data(), d_all, sizeof(double) * res.size(), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    cudaFree(d_all);
    if (e != cudaSuccess) return cuda_fail(e);
    for (int i = 0; i < c->ndirs; ++i) {
        sum_host[i] = res[3 * i];
        if (min_host) min_host[i] = res[3 * i + 1];
        if (max_host) max_host[i] = res[3 * i + 2];
    }
    return RT_OK;
}

extern "C" int rt_direction_records(rt_ctx *c, long long *rec, double *L_host)
{
    if (!c || !rec) return RT_EINVAL;
    for (int i = 0; i < c->ndirs; ++i) {
        const HostDir &h = c->hd[(size_t)i * c->rays * c->rays];
        rec[6 * i + 0] = h.a;
        rec[6 * i + 1] = h.refl[0] | (h.refl[1] << 1) | (h.refl[2] << 2);
        rec[6 * i + 2] = h.Mb;
        rec[6 * i + 3] = h.Mc;
        rec[6 * i + 4] = (c->fast[h.layout] && owned_supported(c->pitch[h.layout], h.Nc, rows_for(c, h.layout), c->nbp)) ? 0 : 1;
        rec[6 * i + 5] = c->rays;
        if (L_host) L_host[i] = h.L;
    }
    return RT_OK;
}

extern "C" int rt_working_set_bytes(rt_ctx *c, unsigned long long *bytes_host)
{
    if (!c || !bytes_host) return RT_EINVAL;
    DevGuard dev_guard(c->device);
    int rc = ensure_buffers(c);
    if (rc != RT_OK) return rc;
    unsigned long long b = 0;
    for (int l = 0; l < 2; ++l) {
        b += sizeof(float2) * (unsigned long long)c->ncell_l[l] * c->nbins;                        // packed fields
        b += 2ull * sizeof(float) * (unsigned long long)c->ncell_l[l] * c->nbins * c->slots[l];   // slot + seam accumulators
    }
    *bytes_host = b;
    return RT_OK;
}

extern "C" int rt_probe_bandwidth(unsigned long long bytes, int mode, int iters, double *gbs_host, void *stream)
{
    if (bytes < (1ull << 20) || bytes > (1ull << 36) || (mode != 0 && mode != 1) || iters < 1 || iters > 1000 || !gbs_host) return RT_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    int dev = 0, sms = 148;
    CK(cudaGetDevice(&dev));
    CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const size_t n4 = (size_t)(bytes / 16);
    float4 *buf = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    cudaError_t e = cudaMalloc(&buf, n4 * 16);
    if (e != cudaSuccess) return e == cudaErrorMemoryAllocation ? RT_ENOMEM : cuda_fail(e);
    if (e == cudaSuccess) e = cudaMemsetAsync(buf, 0, n4 * 16, st);
    if (e == cudaSuccess) e = cudaEventCreate(&e0);
    if (e == cudaSuccess) e = cudaEventCreate(&e1);
    double best = 0.0;
    // enough passes per launch that it lasts of the order of a millisecond (about 8 GB of accesses)
    const int reps = (int)std::max<unsigned long long>(1, std::min<unsigned long long>(512, (8ull << 30) / (n4 * 16)));
    for (int w = 0; w < 2 && e == cudaSuccess; ++w) e = launch_probe(buf, n4, mode, 1, sms, st);   // warm-up: fills L2 if it fits
    for (int i = 0; i < iters && e == cudaSuccess; ++i) {
        e = cudaEventRecord(e0, st);
        if (e == cudaSuccess) e = launch_probe(buf, n4, mode, reps, sms, st);
        if (e == cudaSuccess) e = cudaEventRecord(e1, st);
        if (e == cudaSuccess) e = cudaEventSynchronize(e1);
        float ms = 0.0f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
        if (e == cudaSuccess && ms > 0.0f) best = std::max(best, (double)(n4 * 16) * reps * (mode ? 2.0 : 1.0) / (ms * 1e-3) / 1e9);
    }
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaFree(buf);
    if (e != cudaSuccess) return cuda_fail(e);
    *gbs_host = best;
    return RT_OK;
}

extern "C" int rt_last_launch_count(rt_ctx *c) { return c ? c->last_launches : RT_EINVAL; }

extern "C" int rt_last_sweep_was_graph(rt_ctx *c) { return c ? (c->last_graph ? 1 : 0) : RT_EINVAL; }

extern "C" float rt_last_sweep_kernel_ms(rt_ctx *c)
{
    if (!c || !c->ev_valid) return -1.0f;
    DevGuard dev_guard(c->device);
    if (cudaEventSynchronize(c->ev1) != cudaSuccess) return -1.0f;
    float ms = -1.0f;
    if (cudaEventElapsedTime(&ms, c->ev0, c->ev1) != cudaSuccess) return -1.0f;
    return ms;
}

extern "C" int rt_destroy(rt_ctx *c)
{
    if (!c) return RT_OK;
    DevGuard dev_guard(c->device);
    cudaDeviceSynchronize();
    free_device(c);
    delete c;
    return RT_OK;
}
