// rt_point_sources_static (include/rt.h): RT from point sources (section 2.1; Appendix 1, eqs. A1-A3)
// for callers that must not allocate device memory.
//
// Who that is.  A radiation-hydrodynamics code usually sizes its own arena to nearly all of the GPU's memory at
// start-up and hands out pieces of it; once it has done so, a cudaMalloc made by a library it calls either fails or
// takes memory the host code counted on.  The same holds under a framework's caching allocator (PyTorch's, for
// instance, keeps what it has been given), inside a time step where the device-wide synchronisation that cudaMalloc /
// cudaFree imply would stall every other stream, and on a GPU shared through MPS with a per-client memory limit.
// rt_create, rt_set_fields and rt_point_sources all allocate (tables, packed copies of the fields, accumulators, a
// pinned staging buffer); this entry point allocates nothing, on the device or pinned on the host, ever.
//
// How.  The only memory the point-source kernel needs beyond the caller's kappa and Q (and tau) is (i) a device copy
// of the source tables and (ii) the counter of marched ray pieces.  Both live in ONE array that is part of the
// library image: `rt_static_scratch` below, kScratchBytes = 143,616 bytes, reserved on every GPU on which this library's
// module gets loaded and held until the process exits.  The kernel is k_point_sources (rt_kernels.cu) restated to
// read kappa straight from the caller's [nbins][nz][ny][nx] array (with the same 2^-60 floor the packed copy
// carries) and the luminosities as the caller's fp64 values rounded to fp32 on the fly; per cell it does the same
// operations in the same order, so the two paths agree to rounding (tests/test_zz_no_alloc.py).
//
// What a user has to know (also in rt.h):
//  - capacity: nsrc <= RT_STATIC_MAX_SOURCES (1024), nbins <= RT_STATIC_MAX_BINS (16); beyond -> RT_ELIMIT, nothing enqueued;
//  - the first call on a device looks the array's device address up (cudaGetSymbolAddress, which also makes the
//    CUDA runtime load this file's module on that device); make that first call before any stream capture begins;
//  - every call on a device uses the same array: the source tables of the previous call are overwritten and the
//    counter is cleared on the caller's stream, so two calls whose GPU work overlaps (two streams, two host threads)
//    race on it -- order them (one stream, or an event between them).
#include "../../include/rt.h"
#include "rt_internal.h"

#include <cmath>
#include <mutex>

namespace {

constexpr int kFix = 256;                                  // source positions: 1/256 cell width (rt.h rt_point_sources)
constexpr size_t kOffSteps = 0;                            // unsigned long long: ray pieces marched (atomicAdd target)
constexpr size_t kOffSrc = 256;                            // int32 [RT_STATIC_MAX_SOURCES][3]
constexpr size_t kOffLum = kOffSrc + sizeof(int) * 3 * RT_STATIC_MAX_SOURCES;                 // fp64 [RT_STATIC_MAX_SOURCES][RT_STATIC_MAX_BINS]
constexpr size_t kScratchBytes = kOffLum + sizeof(double) * RT_STATIC_MAX_SOURCES * RT_STATIC_MAX_BINS;
static_assert(kOffLum % 256 == 0 && kScratchBytes == 143616, "scratch layout as documented in rt.h");

// The scratch memory of this file.  In host code this name is only a handle for cudaGetSymbolAddress: it is NOT a
// device address, and a kernel handed `rt_static_scratch` (or &rt_static_scratch[0]) from the host would read and
// write some unrelated host-side shadow or fault.  Host code below only ever uses the pointer scratch_on_device() returns.
static __device__ __align__(256) unsigned char rt_static_scratch[kScratchBytes];

constexpr int kMaxDevices = 64;
std::mutex g_mu;
unsigned char *g_scratch_addr[kMaxDevices];                // device address of rt_static_scratch on device d; null until d's first call

// Set-up, once per device, with that device current: ask the runtime where the array lives on this GPU.
int scratch_on_device(unsigned char **out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return rt::api_cuda_fail(e);
    if (dev < 0 || dev >= kMaxDevices) return RT_EINVAL;
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_scratch_addr[dev]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, rt_static_scratch);
        if (e != cudaSuccess) return rt::api_cuda_fail(e);
        if (!p) return RT_ECUDA;
        g_scratch_addr[dev] = static_cast<unsigned char *>(p);
    }
    *out = g_scratch_addr[dev];
    return RT_OK;
}

// Crossing parameters (exact integers below 2^54): fp64 for meshes up to 512 cells per axis, where they stay below
// 2^52, 64-bit integers above (see rt_kernels.cu).
template <class TT> struct Never;
template <> struct Never<double> { static __device__ __forceinline__ double v() { return 1.0e300; } };
template <> struct Never<long long> { static __device__ __forceinline__ long long v() { return 0x7fffffffffffffffll; } };

template <class TT>
__device__ __forceinline__ void advance(TT &T, int &idx, TT Tn, TT inc, int didx)
{
    if (T == Tn) { idx += didx; T += inc; }
}

// One thread per target cell, one long characteristic per (source, cell) from the source through the cell centre:
//   tau = sum kappa ds over the cells before the target, dtau = kappa_cell (r_out - r_in),
//   Q  += L exp(-tau) (1 - exp(-dtau)) / (4 pi/3 (r_out^3 - r_in^3)).
// src / lum / steps point into rt_static_scratch (passed in: the host resolved the address at set-up).
template <class TT, bool COUNT>
__global__ void __launch_bounds__(128)
k_point_sources_static(float *__restrict__ Q, float *__restrict__ tau_out, const float *__restrict__ kappa,
                       int nx, int ny, int nz, const int *__restrict__ src, const double *__restrict__ lum, int nsrc,
                       int nbins, float cell_width, int diag_src, int diag_bin, unsigned long long *__restrict__ steps)
{
    const int bin = blockIdx.z;
    const long long ncell = (long long)nx * ny * nz;
    const long long cidx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const float *__restrict__ kbin = kappa + (size_t)bin * ncell;
    unsigned nstep = 0;
    if (cidx < ncell) {
        const int tgt[3] = {(int)(cidx % nx), (int)((cidx / nx) % ny), (int)(cidx / ((long long)nx * ny))};
        const int idx_t = (int)cidx;
        const float kap_t = fmaxf(kbin[idx_t], rt::kKappaMin);
        const TT never = Never<TT>::v();
        double q = 0.0;
        for (int a = 0; a < nsrc; ++a) {
            long long s[3], d[3], ad[3];
            TT T[3], inc[3];
            int stp[3], cur[3];
            double len2 = 0.0;
#pragma unroll
            for (int i = 0; i < 3; ++i) {
                s[i] = src[3 * a + i];
                d[i] = ((long long)tgt[i] * kFix + kFix / 2) - s[i];
                stp[i] = d[i] > 0 ? 1 : (d[i] < 0 ? -1 : 0);
                ad[i] = d[i] < 0 ? -d[i] : d[i];
                len2 += (double)d[i] * (double)d[i];
                int c = (int)(s[i] / kFix);
                if (s[i] % kFix == 0 && stp[i] < 0) c -= 1;       // a source on a cell boundary belongs to the cell the ray moves into
                cur[i] = c;
            }
            int idx = (cur[2] * ny + cur[1]) * nx + cur[0];
            const int didx[3] = {stp[0], stp[1] * nx, stp[2] * nx * ny};
            // common denominator |dx dy dz| over the moving axes: T_i = n_i * prod_{j != i} |d_j|
            const long long f0 = ad[0] ? ad[0] : 1, f1 = ad[1] ? ad[1] : 1, f2 = ad[2] ? ad[2] : 1;
            const long long W[3] = {f1 * f2, f0 * f2, f0 * f1};
            const double Dn = (double)f0 * (double)f1 * (double)f2;
            const double len = sqrt(len2) / kFix * (double)cell_width;
            const double scale = len / Dn;                        // length per unit of T
#pragma unroll
            for (int i = 0; i < 3; ++i) {
                if (stp[i] == 0) { T[i] = never; inc[i] = (TT)0; continue; }
                const long long plane = (long long)(cur[i] + (stp[i] > 0 ? 1 : 0)) * kFix;
                T[i] = (TT)((plane - s[i]) * stp[i] * W[i]);
                inc[i] = (TT)((long long)kFix * W[i]);
            }
            double tauT = 0.0, r_in = 0.0, r_out = 0.0, dr = 0.0;
            TT T0 = (TT)0;
            float kap = fmaxf(kbin[idx], rt::kKappaMin);
            for (;;) {
                const TT Tn = T[0] < T[1] ? (T[0] < T[2] ? T[0] : T[2]) : (T[1] < T[2] ? T[1] : T[2]);
                if (COUNT) nstep += 1;
                if (idx == idx_t) {
                    if (Tn == never) { r_in = 0.0; dr = r_out = 0.5 * (double)cell_width; }       // the source sits at this cell's centre
                    else { r_in = (double)T0 * scale; dr = (double)(Tn - T0) * scale; r_out = r_in + dr; }
                    break;
                }
                const double dT = (double)(Tn - T0);
                advance(T[0], idx, Tn, inc[0], didx[0]);          // axes that cross together step together: no zero-length pieces
                advance(T[1], idx, Tn, inc[1], didx[1]);
                advance(T[2], idx, Tn, inc[2], didx[2]);
                tauT = fma((double)kap, dT, tauT);
                kap = fmaxf(kbin[idx], rt::kKappaMin);            // the cell just entered (at the latest the target cell)
                T0 = Tn;
            }
            const double tau = tauT * scale;
            const double dtau = (double)kap_t * dr;
            const double vol = 4.0 * 3.14159265358979323846 / 3.0 * dr * (r_out * r_out + r_out * r_in + r_in * r_in);
            q += (double)(float)lum[(size_t)a * nbins + bin] * exp(-tau) * (-expm1(-dtau)) / vol;
            if (tau_out && a == diag_src && bin == diag_bin) tau_out[cidx] = (float)tau;
        }
        Q[(size_t)bin * ncell + cidx] = (float)q;
    }
    if (COUNT && bin == 0) {
        for (int o = 16; o > 0; o >>= 1) nstep += __shfl_xor_sync(0xffffffffu, nstep, o);
        if ((threadIdx.x & 31) == 0 && nstep) atomicAdd(steps, (unsigned long long)nstep);
    }
}

}  // namespace

#define CKS(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) return rt::api_cuda_fail(e__); } while (0)

extern "C" int rt_point_sources_static(int nx, int ny, int nz, int nbins, double cell_width, const float *kappa_dev,
                                       const int *src_fix_host, const double *lum_host, int nsrc, float *Q_dev,
                                       int diag_src, int diag_bin, float *tau_dev, unsigned long long *steps_host,
                                       void *stream)
{
    if (!kappa_dev || !src_fix_host || !lum_host || !Q_dev) return RT_EINVAL;
    if (nx < 1 || ny < 1 || nz < 1 || nx > 1024 || ny > 1024 || nz > 1024) return RT_EINVAL;   // crossing parameters below 2^54
    if ((long long)nx * ny * nz >= (1ll << 31)) return RT_EINVAL;
    if (nbins < 1 || nsrc < 1 || !(cell_width > 0.0) || !std::isfinite(cell_width)) return RT_EINVAL;
    if (nsrc > RT_STATIC_MAX_SOURCES || nbins > RT_STATIC_MAX_BINS) return RT_ELIMIT;          // the array is only so big
    if (tau_dev && (diag_src < 0 || diag_src >= nsrc || diag_bin < 0 || diag_bin >= nbins)) return RT_EINVAL;
    const int dims[3] = {nx, ny, nz};
    for (int a = 0; a < nsrc; ++a) {
        for (int i = 0; i < 3; ++i)
            if (src_fix_host[3 * a + i] < 0 || src_fix_host[3 * a + i] > dims[i] * kFix) return RT_EINVAL;
        for (int b = 0; b < nbins; ++b) {
            const double v = lum_host[(size_t)a * nbins + b];
            if (!(v >= 0.0) || !std::isfinite(v)) return RT_EINVAL;
        }
    }
    unsigned char *scratch = nullptr;                            // DEVICE address of rt_static_scratch on the current device
    const int rc = scratch_on_device(&scratch);
    if (rc != RT_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    unsigned long long *d_steps = reinterpret_cast<unsigned long long *>(scratch + kOffSteps);
    int *d_src = reinterpret_cast<int *>(scratch + kOffSrc);
    double *d_lum = reinterpret_cast<double *>(scratch + kOffLum);
    // the array still holds the last call's counter and tables: the counter must start at zero, the tables are overwritten
    CKS(cudaMemsetAsync(d_steps, 0, sizeof(unsigned long long), st));
    CKS(cudaMemcpyAsync(d_src, src_fix_host, sizeof(int) * 3 * (size_t)nsrc, cudaMemcpyHostToDevice, st));
    CKS(cudaMemcpyAsync(d_lum, lum_host, sizeof(double) * (size_t)nsrc * nbins, cudaMemcpyHostToDevice, st));
    const long long ncell = (long long)nx * ny * nz;
    const dim3 grid((unsigned)((ncell + 127) / 128), 1, (unsigned)nbins);
    const bool small = nx <= 512 && ny <= 512 && nz <= 512, count = steps_host != nullptr;
#define RT_PSS_LAUNCH(TT, COUNT)                                                                                       \
    k_point_sources_static<TT, COUNT><<<grid, 128, 0, st>>>(Q_dev, tau_dev, kappa_dev, nx, ny, nz, d_src, d_lum, nsrc, nbins, \
                                                           (float)cell_width, diag_src, diag_bin, d_steps)
    if (small) { if (count) RT_PSS_LAUNCH(double, true); else RT_PSS_LAUNCH(double, false); }
    else       { if (count) RT_PSS_LAUNCH(long long, true); else RT_PSS_LAUNCH(long long, false); }
#undef RT_PSS_LAUNCH
    CKS(cudaGetLastError());
    if (steps_host) {                                            // the one synchronising variant: the count comes back to the host
        CKS(cudaMemcpyAsync(steps_host, d_steps, sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
        CKS(cudaStreamSynchronize(st));
    }
    return RT_OK;
}
