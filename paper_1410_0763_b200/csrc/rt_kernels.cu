// sm_100a kernels of the diffuse-radiation ray sweep (arXiv:1410.0763 section 2.2 / 3.1).
//
//   k_build_programs   integer traversal of one slab for all rays of a direction (Fig. 2)
//   k_pack_fields      (kappa, S) -> packed float2 copies: native [z][y][x] and transposed [x][z][y]
//   k_sweep_tma        the hot kernel (rt_sweep.cuh): eq. 7 / eq. 8 per segment, atomic-free J partials by
//                      cell ownership, TMA-staged rows, mirror pairs
//   k_sweep_generic    one thread per lattice ray with per-ray integer traversal; the paper's four
//                      ray groups or atomicAdd -- ablations and fallback
//   k_normalise        eqs. 10-13: sum slot/seam accumulators, 1/(N_d kappa), + S
//   diagnostics        counts finalise, sum-of-ds reduction
//
// See DESIGN.md for the data layout and why the ownership scheme replaces the four ray groups.
#include "rt_internal.h"

#include <algorithm>
#include <type_traits>

namespace rt {

constexpr long long kMaxGridZ = 65535;       // planes (bin, z) per launch of the per-plane kernels; taller stacks loop

// ------------------------------------------------------------------------------------------------
// Slab programs
// ------------------------------------------------------------------------------------------------
__global__ void k_build_programs(const DirDev *__restrict__ dirs, int ndirs, SlabProg *__restrict__ prog,
                                 double cell_width, const double *__restrict__ Lvals)
{
    const int dir = blockIdx.y;
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (dir >= ndirs) return;
    const DirDev D = dirs[dir];
    if (k >= D.Na) return;
    const long long ONE = kOne;
    const long long Mb = D.Mb, Mc = D.Mc;
    // fractional entry position inside the entry cell; the same for every ray of the (sub-)lattice
    // (offsets are whole cells): U = p*ONE + u0 + k*Mb, u0 = ONE/2 for one ray per cell
    const long long u = ((long long)sub_offset(D.sub, 0) + (long long)k * Mb) & (ONE - 1);
    const long long v = ((long long)sub_offset(D.sub, 1) + (long long)k * Mc) & (ONE - 1);
    const long long Db = ONE - u, Dc = ONE - v;          // distance to the next cell boundary, >= 1
    const bool crossb = (u + Mb > ONE), touchb = (u + Mb == ONE);
    const bool crossc = (v + Mc > ONE), touchc = (v + Mc == ONE);
    const double Lw = Lvals[dir] * cell_width;
    const double tb = crossb ? (double)Db / (double)Mb : 1.0;
    const double tc = crossc ? (double)Dc / (double)Mc : 1.0;
    double l0 = 0.0, l1 = 0.0, l2 = 0.0;
    unsigned f = 0;
    if (!crossb && !crossc) {
        l0 = 1.0;
        if (touchb) f |= F_SB1;
        if (touchc) f |= F_SC1;
    } else if (crossb && !crossc) {
        l0 = tb; l1 = 1.0 - tb; f |= F_SB1 | F_P1;
        if (touchc) f |= F_SC2;
    } else if (!crossb && crossc) {
        l0 = tc; l1 = 1.0 - tc; f |= F_SC1 | F_P1;
        if (touchb) f |= F_SB2;
    } else {
        const long long lhs = Db * Mc, rhs = Dc * Mb;     // t_b ? t_c  <=>  Db*Mc ? Dc*Mb  (exact)
        if (lhs < rhs)      { l0 = tb; l1 = tc - tb; l2 = 1.0 - tc; f |= F_SB1 | F_P1 | F_SC2 | F_P2; }
        else if (lhs > rhs) { l0 = tc; l1 = tb - tc; l2 = 1.0 - tb; f |= F_SC1 | F_P1 | F_SB2 | F_P2; }
        else                { l0 = tb; l1 = 1.0 - tb; f |= F_SB1 | F_SC1 | F_P1; }   // diagonal step
    }
    SlabProg s;
    // row shift of the slab (rt_internal.h kShiftBit): whole cells the rays have moved along c before slab k, mod Nc
    const long long shift = (((long long)sub_offset(D.sub, 1) + (long long)k * Mc) >> kF) % D.Nc;
    s.len0 = (float)(l0 * Lw); s.len1 = (float)(l1 * Lw); s.len2 = (float)(l2 * Lw); s.flags = f | ((unsigned)shift << kShiftBit);
    prog[D.prog_off + k] = s;
}

cudaError_t launch_build_programs(const DirDev *dirs, int ndirs, int max_na, SlabProg *prog, double cell_width,
                                  const double *Lvals, cudaStream_t st)
{
    // one thread per (direction, slab): grid.x covers the longest march, grid.y the directions (65535 at most: loop)
    for (int d0 = 0; d0 < ndirs; d0 += 32768) {
        int nd = ndirs - d0 < 32768 ? ndirs - d0 : 32768;
        dim3 grid((max_na + 255) / 256, nd);
        k_build_programs<<<grid, 256, 0, st>>>(dirs + d0, nd, prog, cell_width, Lvals + d0);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

// ------------------------------------------------------------------------------------------------
// Field packing: native copy and (x,y)-transposed copy, kappa floored at kKappaMin
// ------------------------------------------------------------------------------------------------
__global__ void k_pack_fields(const float *__restrict__ kappa, const float *__restrict__ S,
                              float2 *__restrict__ Pnat, float2 *__restrict__ PT, int ppN, int ppT, int nx, int ny, int nz,
                              int nxp, int nyp, int nbp, int zb0)
{
    float *__restrict__ fN = reinterpret_cast<float *>(Pnat);
    float *__restrict__ fT = reinterpret_cast<float *>(PT);
    __shared__ float2 tile[32][33];
    const int zb = (int)blockIdx.z + zb0;                  // (bin, z) planes; grid.z holds at most 65535 of them per launch
    const int bin = zb / nz, z = zb % nz;
    const int x0 = blockIdx.x * 32, y0 = blockIdx.y * 32;
    const size_t ncell = (size_t)nx * ny * nz;
    const size_t boff = (size_t)bin * ncell;
    // rows of the packed copies have pitch nxp / nyp >= nx / ny (pad cells stay zero: kappa = 0 and S = 0
    // leave a ray unchanged and add nothing to an accumulator); bins are planes or packed per row (packed_cell)
    const size_t rowsN = (size_t)ny * nz, rowsT = (size_t)nz * nx;
    for (int dy = threadIdx.y; dy < 32; dy += blockDim.y) {
        int x = x0 + threadIdx.x, y = y0 + dy;
        if (x < nx && y < ny) {
            size_t i = boff + ((size_t)z * ny + y) * nx + x;
            float2 v = make_float2(fmaxf(kappa[i], kKappaMin), S[i]);
            const size_t o = field_index(packed_cell(bin, (size_t)z * ny + y, x, nbp, nxp, rowsN), ppN);
            fN[o] = v.x; fN[o + field_s_offset(ppN)] = v.y;
            tile[dy][threadIdx.x] = v;
        }
    }
    __syncthreads();
    for (int dx = threadIdx.y; dx < 32; dx += blockDim.y) {
        int x = x0 + dx, y = y0 + threadIdx.x;
        if (x < nx && y < ny) {
            const float2 v = tile[threadIdx.x][dx];
            const size_t o = field_index(packed_cell(bin, (size_t)x * nz + z, y, nbp, nyp, rowsT), ppT);
            fT[o] = v.x; fT[o + field_s_offset(ppT)] = v.y;
        }
    }
}

cudaError_t launch_pack_fields(const float *kappa, const float *S, float2 *Pnat, float2 *PT, int ppN, int ppT,
                               int nx, int ny, int nz, int nxp, int nyp, int nbins, int nbp, cudaStream_t st)
{
    const long long planes = (long long)nz * nbins;
    for (long long zb0 = 0; zb0 < planes; zb0 += kMaxGridZ) {
        dim3 grid((nx + 31) / 32, (ny + 31) / 32, (unsigned)std::min<long long>(kMaxGridZ, planes - zb0)), block(32, 8);
        k_pack_fields<<<grid, block, 0, st>>>(kappa, S, Pnat, PT, ppN, ppT, nx, ny, nz, nxp, nyp, nbp, (int)zb0);
        const cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

// ------------------------------------------------------------------------------------------------
// The owned sweep kernel lives in rt_sweep.cuh / rt_sweep_nb*.cu (one translation unit per width).
// ------------------------------------------------------------------------------------------------
cudaError_t launch_sweep_nb32(const SweepLaunch &L, cudaStream_t st);
cudaError_t launch_sweep_nb64(const SweepLaunch &L, cudaStream_t st);
cudaError_t launch_sweep_nb128(const SweepLaunch &L, cudaStream_t st);
cudaError_t launch_sweep_nb256(const SweepLaunch &L, cudaStream_t st);
cudaError_t launch_sweep_nb512(const SweepLaunch &L, cudaStream_t st);
int ctas_per_sm_nb32(int rows, int stages, bool pair);
int ctas_per_sm_nb64(int rows, int stages, bool pair);
int ctas_per_sm_nb128(int rows, int stages, bool pair);
int ctas_per_sm_nb256(int rows, int stages, bool pair);
int ctas_per_sm_nb512(int rows, int stages, bool pair);
// three bins packed per row (rt_sweep_nb*x3.cu)
cudaError_t launch_sweep_nb32x3(const SweepLaunch &L, cudaStream_t st);
cudaError_t launch_sweep_nb64x3(const SweepLaunch &L, cudaStream_t st);
cudaError_t launch_sweep_nb128x3(const SweepLaunch &L, cudaStream_t st);
int ctas_per_sm_nb32x3(int rows, bool pair);
int ctas_per_sm_nb64x3(int rows, bool pair);
int ctas_per_sm_nb128x3(int rows, bool pair);

bool owned_supported(int Nb, int Nc, int rows, int nbp)
{
    if (nbp == 3) return (Nb == 32 || Nb == 64 || Nb == 128) && (rows == 1 || rows == 2) && Nc % rows == 0;
    if (nbp != 1) return false;
    if (!(Nb == 32 || Nb == 64 || Nb == 128 || Nb == 256 || Nb == 512)) return false;
    if (Nb == 512 && rows != 1) return false;
    if (!(rows == 1 || rows == 2 || (rows == 4 && Nb <= 128))) return false;
    return Nc % rows == 0;
}

// resident CTAs (of kOwnedWarpsPerCta warps) per SM of the J-mode owned kernel; 0 if it cannot launch
int owned_ctas_per_sm(int Nb, int rows, int stages, bool pair, int nbp)
{
    if (nbp == 3) {
        switch (Nb) {
        case 32:  return ctas_per_sm_nb32x3(rows, pair);
        case 64:  return ctas_per_sm_nb64x3(rows, pair);
        case 128: return ctas_per_sm_nb128x3(rows, pair);
        }
        return 0;
    }
    switch (Nb) {
    case 32:  return ctas_per_sm_nb32(rows, stages, pair);
    case 64:  return ctas_per_sm_nb64(rows, stages, pair);
    case 128: return ctas_per_sm_nb128(rows, stages, pair);
    case 256: return ctas_per_sm_nb256(rows, stages, pair);
    case 512: return ctas_per_sm_nb512(rows, stages, pair);
    }
    return 0;
}

cudaError_t launch_sweep_owned(const SweepLaunch &L, cudaStream_t st)
{
    if (L.nbp == 3 && L.nbins % 3 == 0) {                  // counting modes run with one bin on plain rows
        switch (L.Nb) {
        case 32:  return launch_sweep_nb32x3(L, st);
        case 64:  return launch_sweep_nb64x3(L, st);
        case 128: return launch_sweep_nb128x3(L, st);
        }
        return cudaErrorInvalidValue;
    }
    switch (L.Nb) {
    case 32:  return launch_sweep_nb32(L, st);
    case 64:  return launch_sweep_nb64(L, st);
    case 128: return launch_sweep_nb128(L, st);
    case 256: return launch_sweep_nb256(L, st);
    case 512: return launch_sweep_nb512(L, st);
    }
    return cudaErrorInvalidValue;
}

// exp / 1 - exp of the generic kernel (same arithmetic as rt_sweep.cuh)
__device__ __forceinline__ float ex2_approx(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float one_minus_exp(float kap, float len, float ct, float &e)
{
    const float x = kap * len;
    const float em = ex2_approx(kap * ct);                     // ct = -len*log2(e)
    float p = fmaf(x, -0.0377338513f, 0.1660640817f);          // x * poly(x) on [0, 1/4], rel. error 3.4e-7
    p = fmaf(x, p, -0.4999701648f);
    p = fmaf(x, p, 0.9999997683f);
    const float ec = fmaf(em, kEx2Bias, em);                   // ex2.approx is biased low (rt_sweep.cuh)
    const float A = x < 0.25f ? x * p : 1.0f - ec;
    e = x < 0.25f ? 1.0f - A : ec;                             // thin pieces: e consistent with A
    return A;
}

// ------------------------------------------------------------------------------------------------
// Generic kernel: one thread per lattice ray, per-ray integer traversal (the paper's own scheme).
//   variant 0: the paper's four ray groups: only rays of L.group march in this
//              launch; their cells are disjoint, so plain read-modify-write is race-free.
//   variant 1: all rays at once with atomicAdd, the measured ablation.
// Works for any mesh dimensions; also the fallback when Nb is not 32/64/128/256.
// ------------------------------------------------------------------------------------------------
template <int MODE>
__global__ void __launch_bounds__(128)
k_sweep_generic(const SweepLaunch L, int np_max, int nq_max)
{
    const int slot = blockIdx.y, bin = blockIdx.z;
    const DirDev D = L.dirs[L.batch[slot]];
    const long long ONE = kOne;
    // extended lattice (reading O3): p from pmin to Nb-1, q from qmin to Nc-1
    const int pmin = -(int)(((long long)D.Na * D.Mb + ONE - 1) / ONE) - 1;
    const int qmin = -(int)(((long long)D.Na * D.Mc + ONE - 1) / ONE) - 1;
    const int np = D.Nb - pmin, nq = D.Nc - qmin;
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (long long)np * nq) return;
    const int p = pmin + (int)(t % np), q = qmin + (int)(t / np);
    if (L.variant == 0) {
        const int g = (((p % 2) + 2) % 2) + 2 * (((q % 2) + 2) % 2);
        if (g != L.group) return;
    }
    const long long foff = (long long)bin * L.ncell + D.base;
    const float *__restrict__ Pf = reinterpret_cast<const float *>(L.P);
    float *acc = L.acc + ((long long)slot * L.nbins) * L.ncell + foff;
    const float invL = (MODE == MODE_J) ? D.invL : 1.0f;
    const int rr = (D.sub >> 16) > 0 ? (D.sub >> 16) : 1;
    const float Lw = 1.0f / (D.invL * (float)(rr * rr));              // slab length L * cell_width (invL carries 1 / r^2)
    const bool rev = D.sj < 0;
    const long long U0 = (long long)p * ONE + sub_offset(D.sub, 0), V0 = (long long)q * ONE + sub_offset(D.sub, 1);
    // inflow of the face the ray enters through = the face it crosses last: the a-face if it starts inside
    // the transverse extent, else the side face whose plane it reaches later (both at once: c)
    float I;
    {
        const int fa = (D.layout >> 8) & 7, fb = (D.layout >> 12) & 7, fc = (D.layout >> 16) & 7;
        const bool inb = U0 >= 0, inc = V0 >= 0;
        int f;
        if (inb && inc) f = fa;
        else if (inb) f = fc;
        else if (inc) f = fb;
        else f = ((-V0) * (long long)D.Mb >= (-U0) * (long long)D.Mc) ? fc : fb;
        I = L.Ibc[6 * bin + f];
    }
    for (int k = 0; k < D.Na; ++k) {
        const long long U = U0 + (long long)k * D.Mb, V = V0 + (long long)k * D.Mc;
        const long long j = U >> kF, l = V >> kF;
        if (j < -1 || j >= D.Nb || l < -1 || l >= D.Nc) continue;
        const long long Db = (j + 1) * ONE - U, Dc = (l + 1) * ONE - V;
        const bool crossb = (U + D.Mb > (j + 1) * ONE), crossc = (V + D.Mc > (l + 1) * ONE);
        float tt[4];
        int dj[3], dl[3], n = 0;
        tt[0] = 0.0f;
        const float tb = crossb ? (float)Db / (float)D.Mb : 1.0f;
        const float tc = crossc ? (float)Dc / (float)D.Mc : 1.0f;
        bool mid = true;
        if (!crossb && !crossc) { dj[0] = 0; dl[0] = 0; tt[1] = 1.0f; n = 1; }
        else if (crossb && !crossc) { dj[0] = 0; dl[0] = 0; tt[1] = tb; dj[1] = 1; dl[1] = 0; tt[2] = 1.0f; n = 2; }
        else if (!crossb && crossc) { dj[0] = 0; dl[0] = 0; tt[1] = tc; dj[1] = 0; dl[1] = 1; tt[2] = 1.0f; n = 2; }
        else {
            const long long lhs = Db * D.Mc, rhs = Dc * D.Mb;
            if (lhs < rhs)      { dj[0] = 0; dl[0] = 0; tt[1] = tb; dj[1] = 1; dl[1] = 0; tt[2] = tc; dj[2] = 1; dl[2] = 1; tt[3] = 1.0f; n = 3; }
            else if (lhs > rhs) { dj[0] = 0; dl[0] = 0; tt[1] = tc; dj[1] = 0; dl[1] = 1; tt[2] = tb; dj[2] = 1; dl[2] = 1; tt[3] = 1.0f; n = 3; }
            else                { dj[0] = 0; dl[0] = 0; tt[1] = tb; dj[1] = 1; dl[1] = 1; tt[2] = 1.0f; n = 2; mid = false; }
        }
        (void)mid;
        for (int s = 0; s < n; ++s) {
            const long long jj = j + dj[s], ll = l + dl[s];
            if (jj < 0 || jj >= D.Nb || ll < 0 || ll >= D.Nc) continue;
            // existence of a piece is an integer fact (exact): first and last pieces always have positive
            // length; the middle piece of a 3-piece slab exists because lhs != rhs there
            const float len = (tt[s + 1] - tt[s]) * Lw;
            const long long o = (long long)k * D.sk + ll * D.sl + (rev ? (D.Nb - 1 - jj) : jj);
            float v = 0.0f;
            if (MODE == MODE_J) {
                const size_t fo = field_index((size_t)(foff + o), L.pp);
                const float2 ks = make_float2(Pf[fo], Pf[fo + field_s_offset(L.pp)]);
                float e;
                const float A = one_minus_exp(ks.x, len, -len * 1.4426950408889634f, e);
                v = I * A * invL;
                I = fmaf(I, e, ks.y * A);
            } else if (MODE == MODE_COUNT) {
                v = 1.0f;
            } else {
                v = len;
            }
            if (L.variant == 1) atomicAdd(acc + o, v);
            else acc[o] += v;
        }
    }
}

cudaError_t launch_sweep_generic(const SweepLaunch &L, int np_max, int nq_max, cudaStream_t st)
{
    const long long nrays = (long long)np_max * nq_max;
    dim3 grid((unsigned)((nrays + 127) / 128), L.nslots, L.nbins), block(128);
    switch (L.mode) {
    case MODE_J:     k_sweep_generic<MODE_J><<<grid, block, 0, st>>>(L, np_max, nq_max); break;
    case MODE_COUNT: k_sweep_generic<MODE_COUNT><<<grid, block, 0, st>>>(L, np_max, nq_max); break;
    default:         k_sweep_generic<MODE_DS><<<grid, block, 0, st>>>(L, np_max, nq_max); break;
    }
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// Normalisation (eqs. 10-13) and diagnostics finalisation.
// Sums the slot and seam accumulators of the native layout and, through a shared-memory tile
// transpose, of the transposed layout.
// ------------------------------------------------------------------------------------------------
template <bool COUNTS> __device__ __forceinline__ typename std::conditional<COUNTS, unsigned long long, double>::type widen(float v);
template <> __device__ __forceinline__ unsigned long long widen<true>(float v) { return (unsigned long long)__float2uint_rn(v); }
template <> __device__ __forceinline__ double widen<false>(float v) { return (double)v; }

// sum over the slots of (slot accumulator + seam accumulator) of one cell: eight independent loads per step (four
// slots) so that enough bytes are in flight per SM to keep HBM busy (the kernel reads every slot of both layouts once:
// 4 GB at C4), with streaming loads (nothing is read twice); a 32^3 mesh is all latency here
template <bool COUNTS>
__device__ __forceinline__ typename std::conditional<COUNTS, unsigned long long, double>::type
sum_slots(const float *__restrict__ acc, const float *__restrict__ accC, int slots, size_t stride, size_t i)
{
    typename std::conditional<COUNTS, unsigned long long, double>::type s0 = 0, s1 = 0, s2 = 0, s3 = 0;
    const float *__restrict__ pa = acc + i, *__restrict__ pc = accC + i;
    int sl = 0;
    for (; sl + 3 < slots; sl += 4, pa += 4 * stride, pc += 4 * stride) {
        const float a0 = __ldcs(pa), c0 = __ldcs(pc), a1 = __ldcs(pa + stride), c1 = __ldcs(pc + stride);
        const float a2 = __ldcs(pa + 2 * stride), c2 = __ldcs(pc + 2 * stride), a3 = __ldcs(pa + 3 * stride), c3 = __ldcs(pc + 3 * stride);
        s0 += widen<COUNTS>(a0); s1 += widen<COUNTS>(c0); s2 += widen<COUNTS>(a1); s3 += widen<COUNTS>(c1);
        s0 += widen<COUNTS>(a2); s1 += widen<COUNTS>(c2); s2 += widen<COUNTS>(a3); s3 += widen<COUNTS>(c3);
    }
    for (; sl < slots; ++sl, pa += stride, pc += stride) { s0 += widen<COUNTS>(__ldcs(pa)); s1 += widen<COUNTS>(__ldcs(pc)); }
    return (s0 + s1) + (s2 + s3);
}

template <bool COUNTS>
__global__ void __launch_bounds__(1024) k_finalise(float *__restrict__ J, unsigned *__restrict__ counts, const float2 *__restrict__ Pnat, int ppN,
                           const float *__restrict__ accN, const float *__restrict__ accNC, int slotsN,
                           const float *__restrict__ accT, const float *__restrict__ accTC, int slotsT,
                           int nx, int ny, int nz, int nxp, int nyp, int nbins, int nbp, float inv_nd, int add_S, int zb0)
{
    using SumT = typename std::conditional<COUNTS, unsigned long long, double>::type;
    __shared__ SumT tile[32][33];
    const int zb = (int)blockIdx.z + zb0;
    const int bin = zb / nz, z = zb % nz;
    const int x0 = blockIdx.x * 32, y0 = blockIdx.y * 32;
    const size_t ncell = (size_t)nx * ny * nz;
    const size_t ncellN = (size_t)nxp * ny * nz, ncellT = (size_t)nyp * nz * nx;      // padded row pitch per layout
    const size_t strideN = ncellN * nbins, strideT = ncellT * nbins;
    // The slot partials are summed in fp64 (J) or as integers (counts: every slot partial is an exact integer below
    // 2^24, rt_create bounds 3 N_d r^2): the kernel is bound by its loads, and the sum over up to a few hundred slot
    // and seam partials then adds no rounding of its own to J.
    // transposed layout [x][z][y]: coalesced along y
    for (int dx = threadIdx.y; dx < 32; dx += blockDim.y) {
        const int x = x0 + dx, y = y0 + threadIdx.x;
        SumT s = 0;
        if (x < nx && y < ny) {
            const size_t i = packed_cell(bin, (size_t)x * nz + z, y, nbp, nyp, (size_t)nz * nx);
            s = sum_slots<COUNTS>(accT, accTC, slotsT, strideT, i);
        }
        tile[dx][threadIdx.x] = s;
    }
    __syncthreads();
    for (int dy = threadIdx.y; dy < 32; dy += blockDim.y) {
        const int x = x0 + threadIdx.x, y = y0 + dy;
        if (x < nx && y < ny) {
            const size_t i = (size_t)bin * ncell + ((size_t)z * ny + y) * nx + x;
            const size_t ip = packed_cell(bin, (size_t)z * ny + y, x, nbp, nxp, (size_t)ny * nz);
            const SumT s = tile[threadIdx.x][dy] + sum_slots<COUNTS>(accN, accNC, slotsN, strideN, ip);
            if (COUNTS) {
                counts[i] = (unsigned)s;
            } else {
                const float *__restrict__ fN = reinterpret_cast<const float *>(Pnat);
                const size_t o = field_index(ip, ppN);
                const float2 ks = make_float2(fN[o], fN[o + field_s_offset(ppN)]);
                const float jin = (float)(s * (double)inv_nd) / ks.x;
                J[i] = add_S ? jin + ks.y : jin;
            }
        }
    }
}

// Two adjacent cells per thread (float2 streaming loads, 64 x 64 tiles): every warp access is a 256-byte run of one
// accumulator row instead of 128 bytes, which is what the DRAM pages want when 2 x (slotsN + slotsT) arrays are read
// side by side (the 32 x 32 form reads the 4 GB of C4 at 3.1 TB/s).  Same arithmetic per cell, in the same order,
// as k_finalise<false>.  Needs even nx and ny (the row pitches always are).
__device__ __forceinline__ void sum_slots2(const float *__restrict__ acc, const float *__restrict__ accC, int slots, size_t stride,
                                           size_t i, double &r0, double &r1)
{
    double a0 = 0, a1 = 0, a2 = 0, a3 = 0, b0 = 0, b1 = 0, b2 = 0, b3 = 0;       // the four partial sums of sum_slots, per cell
    const float2 *__restrict__ pa = reinterpret_cast<const float2 *>(acc + i), *__restrict__ pc = reinterpret_cast<const float2 *>(accC + i);
    const size_t st2 = stride / 2;                                               // stride (cells per slot) is even
    int sl = 0;
    for (; sl + 3 < slots; sl += 4, pa += 4 * st2, pc += 4 * st2) {
        const float2 u0 = __ldcs(pa), v0 = __ldcs(pc), u1 = __ldcs(pa + st2), v1 = __ldcs(pc + st2);
        const float2 u2 = __ldcs(pa + 2 * st2), v2 = __ldcs(pc + 2 * st2), u3 = __ldcs(pa + 3 * st2), v3 = __ldcs(pc + 3 * st2);
        a0 += (double)u0.x; a1 += (double)v0.x; a2 += (double)u1.x; a3 += (double)v1.x;
        a0 += (double)u2.x; a1 += (double)v2.x; a2 += (double)u3.x; a3 += (double)v3.x;
        b0 += (double)u0.y; b1 += (double)v0.y; b2 += (double)u1.y; b3 += (double)v1.y;
        b0 += (double)u2.y; b1 += (double)v2.y; b2 += (double)u3.y; b3 += (double)v3.y;
    }
    for (; sl < slots; ++sl, pa += st2, pc += st2) {
        const float2 u = __ldcs(pa), v = __ldcs(pc);
        a0 += (double)u.x; a1 += (double)v.x; b0 += (double)u.y; b1 += (double)v.y;
    }
    r0 = (a0 + a1) + (a2 + a3);
    r1 = (b0 + b1) + (b2 + b3);
}

__global__ void __launch_bounds__(1024) k_finalise_wide(float *__restrict__ J, const float2 *__restrict__ Pnat, int ppN,
                           const float *__restrict__ accN, const float *__restrict__ accNC, int slotsN,
                           const float *__restrict__ accT, const float *__restrict__ accTC, int slotsT,
                           int nx, int ny, int nz, int nxp, int nyp, int nbins, int nbp, float inv_nd, int add_S, int zb0)
{
    __shared__ double tile[64][65];
    const int zb = (int)blockIdx.z + zb0;
    const int bin = zb / nz, z = zb % nz;
    const int x0 = blockIdx.x * 64, y0 = blockIdx.y * 64;
    const size_t ncell = (size_t)nx * ny * nz;
    const size_t ncellN = (size_t)nxp * ny * nz, ncellT = (size_t)nyp * nz * nx;
    const size_t strideN = ncellN * nbins, strideT = ncellT * nbins;
    // transposed layout [x][z][y]: two adjacent y per thread
    for (int dx = threadIdx.y; dx < 64; dx += 32) {
        const int x = x0 + dx, y = y0 + 2 * (int)threadIdx.x;
        double s0 = 0.0, s1 = 0.0;
        if (x < nx && y < ny)
            sum_slots2(accT, accTC, slotsT, strideT, packed_cell(bin, (size_t)x * nz + z, y, nbp, nyp, (size_t)nz * nx), s0, s1);
        tile[dx][2 * threadIdx.x] = s0;
        tile[dx][2 * threadIdx.x + 1] = s1;
    }
    __syncthreads();
    const float *__restrict__ fN = reinterpret_cast<const float *>(Pnat);
    for (int dy = threadIdx.y; dy < 64; dy += 32) {
        const int x = x0 + 2 * (int)threadIdx.x, y = y0 + dy;
        if (x < nx && y < ny) {
            const size_t ip = packed_cell(bin, (size_t)z * ny + y, x, nbp, nxp, (size_t)ny * nz);
            double n0, n1;
            sum_slots2(accN, accNC, slotsN, strideN, ip, n0, n1);
            const double s0 = tile[2 * threadIdx.x][dy] + n0, s1 = tile[2 * threadIdx.x + 1][dy] + n1;
            // (kappa, S) of the two cells: one 16-byte load in either packed form (rt_internal.h field_index; ip is even)
            const float4 f = *reinterpret_cast<const float4 *>(fN + 2 * ip);
            const float k0 = f.x, k1 = ppN ? f.y : f.z, S0 = ppN ? f.z : f.y, S1 = f.w;
            const float j0 = (float)(s0 * (double)inv_nd) / k0, j1 = (float)(s1 * (double)inv_nd) / k1;
            const size_t i = (size_t)bin * ncell + ((size_t)z * ny + y) * nx + x;
            *reinterpret_cast<float2 *>(J + i) = make_float2(add_S ? j0 + S0 : j0, add_S ? j1 + S1 : j1);
        }
    }
}

cudaError_t launch_normalise(float *J, const float2 *Pnat, int ppN, const float *accN, const float *accNC, int slotsN,
                             const float *accT, const float *accTC, int slotsT,
                             int nx, int ny, int nz, int nxp, int nyp, int nbins, int nbp, float inv_nd, int add_S, cudaStream_t st)
{
    const long long planes = (long long)nz * nbins;
    const bool wide = nx % 2 == 0 && ny % 2 == 0 && nx >= 128 && ny >= 128 && (reinterpret_cast<uintptr_t>(J) & 7u) == 0;
    for (long long zb0 = 0; zb0 < planes; zb0 += kMaxGridZ) {
        if (wide) {
            dim3 grid((nx + 63) / 64, (ny + 63) / 64, (unsigned)std::min<long long>(kMaxGridZ, planes - zb0)), block(32, 32);
            k_finalise_wide<<<grid, block, 0, st>>>(J, Pnat, ppN, accN, accNC, slotsN, accT, accTC, slotsT,
                                                    nx, ny, nz, nxp, nyp, nbins, nbp, inv_nd, add_S, (int)zb0);
            const cudaError_t e = cudaGetLastError();
            if (e != cudaSuccess) return e;
            continue;
        }
        dim3 grid((nx + 31) / 32, (ny + 31) / 32, (unsigned)std::min<long long>(kMaxGridZ, planes - zb0)), block(32, 32);
        k_finalise<false><<<grid, block, 0, st>>>(J, nullptr, Pnat, ppN, accN, accNC, slotsN, accT, accTC, slotsT,
                                                  nx, ny, nz, nxp, nyp, nbins, nbp, inv_nd, add_S, (int)zb0);
        const cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

// ------------------------------------------------------------------------------------------------
// Rates epilogue (eqs. 14-15 with the rectangular bins of eqs. 22-23; eqs. 20-21 are its one-bin case):
//   Gamma = sum_b wG[b] * J_in[b] + lG[b] * S[b],   Heat = sum_b wH[b] * J_in[b] + lH[b] * S[b]
// fused with the normalisation (the accumulators are read once, J is never written).
// ------------------------------------------------------------------------------------------------
struct RateWeights { float wG[16], lG[16], wH[16], lH[16]; };

__global__ void k_rates(float *__restrict__ Gamma, float *__restrict__ Heat, const float2 *__restrict__ Pnat, int ppN,
                        const float *__restrict__ accN, const float *__restrict__ accNC, int slotsN,
                        const float *__restrict__ accT, const float *__restrict__ accTC, int slotsT,
                        int nx, int ny, int nz, int nxp, int nyp, int nbins, int nbp, float inv_nd, const RateWeights W, int z0)
{
    __shared__ double tile[32][33];
    const int z = (int)blockIdx.z + z0;
    const int x0 = blockIdx.x * 32, y0 = blockIdx.y * 32;
    const size_t ncellN = (size_t)nxp * ny * nz, ncellT = (size_t)nyp * nz * nx;
    const size_t strideN = ncellN * nbins, strideT = ncellT * nbins;
    const float *__restrict__ fN = reinterpret_cast<const float *>(Pnat);
    float g[4] = {0.0f, 0.0f, 0.0f, 0.0f}, h[4] = {0.0f, 0.0f, 0.0f, 0.0f};      // rows threadIdx.y + 8 j
    for (int bin = 0; bin < nbins; ++bin) {
        // transposed layout [x][z][y]: coalesced along y
        for (int dx = threadIdx.y; dx < 32; dx += blockDim.y) {
            const int x = x0 + dx, y = y0 + threadIdx.x;
            double s = 0.0;
            if (x < nx && y < ny) {
                const size_t i = packed_cell(bin, (size_t)x * nz + z, y, nbp, nyp, (size_t)nz * nx);
                s = sum_slots<false>(accT, accTC, slotsT, strideT, i);
            }
            tile[dx][threadIdx.x] = s;
        }
        __syncthreads();
        int j = 0;
        for (int dy = threadIdx.y; dy < 32; dy += blockDim.y, ++j) {
            const int x = x0 + threadIdx.x, y = y0 + dy;
            if (x < nx && y < ny) {
                const size_t i = packed_cell(bin, (size_t)z * ny + y, x, nbp, nxp, (size_t)ny * nz);
                const double s = tile[threadIdx.x][dy] + sum_slots<false>(accN, accNC, slotsN, strideN, i);
                const size_t o = field_index(i, ppN);
                const float kap = fN[o], src = fN[o + field_s_offset(ppN)];
                const float jin = (float)(s * (double)inv_nd) / kap;
                g[j] = fmaf(W.wG[bin], jin, fmaf(W.lG[bin], src, g[j]));
                h[j] = fmaf(W.wH[bin], jin, fmaf(W.lH[bin], src, h[j]));
            }
        }
        __syncthreads();
    }
    int j = 0;
    for (int dy = threadIdx.y; dy < 32; dy += blockDim.y, ++j) {
        const int x = x0 + threadIdx.x, y = y0 + dy;
        if (x < nx && y < ny) {
            const size_t i = ((size_t)z * ny + y) * nx + x;
            Gamma[i] = g[j];
            Heat[i] = h[j];
        }
    }
}

// k_rates with two adjacent cells per thread and 64 x 64 tiles (see k_finalise_wide): same arithmetic per cell
__global__ void __launch_bounds__(1024) k_rates_wide(float *__restrict__ Gamma, float *__restrict__ Heat, const float2 *__restrict__ Pnat, int ppN,
                        const float *__restrict__ accN, const float *__restrict__ accNC, int slotsN,
                        const float *__restrict__ accT, const float *__restrict__ accTC, int slotsT,
                        int nx, int ny, int nz, int nxp, int nyp, int nbins, int nbp, float inv_nd, const RateWeights W, int z0)
{
    __shared__ double tile[64][65];
    const int z = (int)blockIdx.z + z0;
    const int x0 = blockIdx.x * 64, y0 = blockIdx.y * 64;
    const size_t ncellN = (size_t)nxp * ny * nz, ncellT = (size_t)nyp * nz * nx;
    const size_t strideN = ncellN * nbins, strideT = ncellT * nbins;
    const float *__restrict__ fN = reinterpret_cast<const float *>(Pnat);
    float g[2][2] = {{0.0f, 0.0f}, {0.0f, 0.0f}}, h[2][2] = {{0.0f, 0.0f}, {0.0f, 0.0f}};      // [row ty + 32 j][cell]
    for (int bin = 0; bin < nbins; ++bin) {
        for (int dx = threadIdx.y; dx < 64; dx += 32) {
            const int x = x0 + dx, y = y0 + 2 * (int)threadIdx.x;
            double s0 = 0.0, s1 = 0.0;
            if (x < nx && y < ny)
                sum_slots2(accT, accTC, slotsT, strideT, packed_cell(bin, (size_t)x * nz + z, y, nbp, nyp, (size_t)nz * nx), s0, s1);
            tile[dx][2 * threadIdx.x] = s0;
            tile[dx][2 * threadIdx.x + 1] = s1;
        }
        __syncthreads();
        int j = 0;
        for (int dy = threadIdx.y; dy < 64; dy += 32, ++j) {
            const int x = x0 + 2 * (int)threadIdx.x, y = y0 + dy;
            if (x < nx && y < ny) {
                const size_t ip = packed_cell(bin, (size_t)z * ny + y, x, nbp, nxp, (size_t)ny * nz);
                double n0, n1;
                sum_slots2(accN, accNC, slotsN, strideN, ip, n0, n1);
                const double s0 = tile[2 * threadIdx.x][dy] + n0, s1 = tile[2 * threadIdx.x + 1][dy] + n1;
                const float4 f = *reinterpret_cast<const float4 *>(fN + 2 * ip);
                const float k0 = f.x, k1 = ppN ? f.y : f.z, S0 = ppN ? f.z : f.y, S1 = f.w;
                const float j0 = (float)(s0 * (double)inv_nd) / k0, j1 = (float)(s1 * (double)inv_nd) / k1;
                g[j][0] = fmaf(W.wG[bin], j0, fmaf(W.lG[bin], S0, g[j][0]));
                g[j][1] = fmaf(W.wG[bin], j1, fmaf(W.lG[bin], S1, g[j][1]));
                h[j][0] = fmaf(W.wH[bin], j0, fmaf(W.lH[bin], S0, h[j][0]));
                h[j][1] = fmaf(W.wH[bin], j1, fmaf(W.lH[bin], S1, h[j][1]));
            }
        }
        __syncthreads();
    }
    int j = 0;
    for (int dy = threadIdx.y; dy < 64; dy += 32, ++j) {
        const int x = x0 + 2 * (int)threadIdx.x, y = y0 + dy;
        if (x < nx && y < ny) {
            const size_t i = ((size_t)z * ny + y) * nx + x;
            *reinterpret_cast<float2 *>(Gamma + i) = make_float2(g[j][0], g[j][1]);
            *reinterpret_cast<float2 *>(Heat + i) = make_float2(h[j][0], h[j][1]);
        }
    }
}

cudaError_t launch_rates(float *Gamma, float *Heat, const float2 *Pnat, int ppN, const float *accN, const float *accNC,
                         int slotsN, const float *accT, const float *accTC, int slotsT, int nx, int ny, int nz,
                         int nxp, int nyp, int nbins, int nbp,
                         float inv_nd, const float *w4 /* host: wG, lG, wH, lH, each [nbins] */, cudaStream_t st)
{
    RateWeights W;
    for (int b = 0; b < 16; ++b) {
        const bool in = b < nbins;
        W.wG[b] = in ? w4[b] : 0.0f;             W.lG[b] = in ? w4[nbins + b] : 0.0f;
        W.wH[b] = in ? w4[2 * nbins + b] : 0.0f; W.lH[b] = in ? w4[3 * nbins + b] : 0.0f;
    }
    const bool wide = nx % 2 == 0 && ny % 2 == 0 && nx >= 128 && ny >= 128 &&
                      ((reinterpret_cast<uintptr_t>(Gamma) | reinterpret_cast<uintptr_t>(Heat)) & 7u) == 0;
    for (long long z0 = 0; z0 < nz; z0 += kMaxGridZ) {
        if (wide) {
            dim3 grid((nx + 63) / 64, (ny + 63) / 64, (unsigned)std::min<long long>(kMaxGridZ, nz - z0)), block(32, 32);
            k_rates_wide<<<grid, block, 0, st>>>(Gamma, Heat, Pnat, ppN, accN, accNC, slotsN, accT, accTC, slotsT, nx, ny, nz, nxp, nyp,
                                                nbins, nbp, inv_nd, W, (int)z0);
            const cudaError_t e = cudaGetLastError();
            if (e != cudaSuccess) return e;
            continue;
        }
        dim3 grid((nx + 31) / 32, (ny + 31) / 32, (unsigned)std::min<long long>(kMaxGridZ, nz - z0)), block(32, 8);
        k_rates<<<grid, block, 0, st>>>(Gamma, Heat, Pnat, ppN, accN, accNC, slotsN, accT, accTC, slotsT, nx, ny, nz, nxp, nyp,
                                       nbins, nbp, inv_nd, W, (int)z0);
        const cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

// ------------------------------------------------------------------------------------------------
// Combine step of a direction-sharded sweep: the un-normalised sums of all
// shards have been added (all-reduce); J_in = sum / N_d (eq. 13), J = J_in + S (eq. 12).
// ------------------------------------------------------------------------------------------------
__global__ void k_combine(float *__restrict__ J, const float *__restrict__ sum, const float2 *__restrict__ Pnat, int ppN,
                          size_t n, int nx, int ny, int nz, int nxp, int nbp, float inv_nd, int add_S)
{
    const float *__restrict__ fN = reinterpret_cast<const float *>(Pnat);
    const size_t rows = (size_t)ny * nz;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        float v = sum[i] * inv_nd;
        if (add_S) {
            const size_t r = i / nx;                               // (bin, z, y) of the caller's [nbins][nz][ny][nx] array
            const size_t ip = packed_cell((int)(r / rows), r % rows, (int)(i % nx), nbp, nxp, rows);
            v += fN[field_index(ip, ppN) + field_s_offset(ppN)];
        }
        J[i] = v;
    }
}

cudaError_t launch_combine(float *J, const float *sum, const float2 *Pnat, int ppN, int nx, int ny, int nz, int nxp,
                           int nbins, int nbp, float inv_nd, int add_S, cudaStream_t st)
{
    const size_t n = (size_t)nx * ny * nz * nbins;
    size_t blocks = (n + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    k_combine<<<(unsigned)blocks, 256, 0, st>>>(J, sum, Pnat, ppN, n, nx, ny, nz, nxp, nbp, inv_nd, add_S);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// Point radiation sources (section 2.1; Appendix 1 eqs. A1-A3): one thread per target
// cell, one long characteristic per (source, cell) from the source through the cell centre.
//   tau  = sum kappa ds over the cells before the target cell, dtau = kappa_cell (r_out - r_in)
//   Q   += L exp(-tau) (1 - exp(-dtau)) / (4 pi/3 (r_out^3 - r_in^3))
// Source positions are integers in units of 1/256 cell, so every traversal decision is exact: the
// crossing parameters of the three axes are compared on the common denominator |dx dy dz| in 64-bit
// integers (u_i = T_i / Dn, one add per step); axes that cross together step together and
// zero-length pieces are dropped.  Threads of a warp hold 32 neighbouring cells of a row: their rays
// from one source are nearly parallel, so the kappa gathers of a warp fall into a few cache lines.
// ------------------------------------------------------------------------------------------------
constexpr int kPsFix = 256;

// Crossing parameters T_i (position along the ray in units of 1 / |dx dy dz|) are exact integers below 2^54.  For
// meshes up to 512 cells per axis they stay below 2^52 and are held in fp64 (TT = double): every add, compare and
// difference is exact there too, and costs one instruction instead of the two to three a 64-bit integer takes on
// the 32-bit ALU.  Larger meshes (up to 1024) use 64-bit integers.
template <class TT> struct PsInf;
template <> struct PsInf<double> { static __device__ __forceinline__ double v() { return 1.0e300; } };
template <> struct PsInf<long long> { static __device__ __forceinline__ long long v() { return 0x7fffffffffffffffll; } };

// plain minimum (no NaN handling: the operands are exact integers or the "never" marker)
template <class TT> __device__ __forceinline__ TT ps_min(TT a, TT b) { return a < b ? a : b; }
// one axis of a ray step: if this axis' next plane is the one reached (T == Tn), move to the next cell along it and
// schedule its next plane.  Predicated adds instead of selects: three instructions per axis.
__device__ __forceinline__ void ps_advance(double &T, int &idx, double Tn, double inc, int didx)
{
    asm("{\n\t.reg .pred p;\n\tsetp.eq.f64 p, %0, %2;\n\t@p add.f64 %0, %0, %3;\n\t@p add.s32 %1, %1, %4;\n\t}"
        : "+d"(T), "+r"(idx) : "d"(Tn), "d"(inc), "r"(didx));
}
__device__ __forceinline__ void ps_advance(long long &T, int &idx, long long Tn, long long inc, int didx)
{
    if (T == Tn) { idx += didx; T += inc; }
}

// PP: the packed native copy is pair-packed (a compile-time constant keeps its index arithmetic out of the ray step);
// COUNT: the step count is wanted (the parity gate), else the counter is not kept
template <class TT, int PP, bool COUNT>
__global__ void __launch_bounds__(128)
k_point_sources(float *__restrict__ Q, float *__restrict__ tau_out, const float2 *__restrict__ Pnat, int ppN_,
                int nx, int ny, int nz, int nxp, const int *__restrict__ src, const float *__restrict__ lum, int nsrc,
                int nbins, int nbp, float cell_width, int diag_src, int diag_bin, unsigned long long *__restrict__ steps)
{
    constexpr int ppN = PP;
    (void)ppN_;
    const int bin = blockIdx.z;
    const long long ncell = (long long)nx * ny * nz;
    const long long cidx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const bool live = cidx < ncell;
    const float *__restrict__ fN = reinterpret_cast<const float *>(Pnat);
    // this bin's cells in the packed native copy: cell (row, x) at boffN + row * rowp + x (packed_cell: bins are planes,
    // or nbp bins share a row)
    const size_t boffN = packed_cell(bin, 0, 0, nbp, nxp, (size_t)ny * nz);
    const int rowp = nxp * nbp;
    unsigned nstep = 0;
    if (live) {
        const int tgt[3] = {(int)(cidx % nx), (int)((cidx / nx) % ny), (int)(cidx / ((long long)nx * ny))};
        const float kap_t = fN[field_index(boffN + ((size_t)tgt[2] * ny + tgt[1]) * rowp + tgt[0], ppN)];
        const float *__restrict__ fbin = fN + 2 * boffN;          // this bin's cells of the packed copy (boffN is even: nxp is)
        double q = 0.0;
        // linear index of a cell in the packed native copy (row pitch nxp) and its change per step along an axis
        const int idx_t = (tgt[2] * ny + tgt[1]) * rowp + tgt[0];
        const TT kInf = PsInf<TT>::v();
        for (int a = 0; a < nsrc; ++a) {
            long long s[3], d[3], ad[3];
            TT T[3], inc[3];
            int stp[3], cur[3];
            double len2 = 0.0;
#pragma unroll
            for (int i = 0; i < 3; ++i) {
                s[i] = src[3 * a + i];
                d[i] = ((long long)tgt[i] * kPsFix + kPsFix / 2) - s[i];
                stp[i] = d[i] > 0 ? 1 : (d[i] < 0 ? -1 : 0);
                ad[i] = d[i] < 0 ? -d[i] : d[i];
                len2 += (double)d[i] * (double)d[i];
                int c = (int)(s[i] / kPsFix);
                if (s[i] % kPsFix == 0 && stp[i] < 0) c -= 1;     // a source on a boundary belongs to the cell the ray moves into
                cur[i] = c;
            }
            int idx = (cur[2] * ny + cur[1]) * rowp + cur[0];
            const int didx[3] = {stp[0], stp[1] * rowp, stp[2] * rowp * ny};
            // common denominator over the moving axes; T_i = n_i * prod_{j != i} |d_j|
            const long long f0 = ad[0] ? ad[0] : 1, f1 = ad[1] ? ad[1] : 1, f2 = ad[2] ? ad[2] : 1;
            const long long W[3] = {f1 * f2, f0 * f2, f0 * f1};
            const double Dn = (double)f0 * (double)f1 * (double)f2;
            const double len = sqrt(len2) / kPsFix * (double)cell_width;
            const double scale = len / Dn;                          // length per unit of T
#pragma unroll
            for (int i = 0; i < 3; ++i) {
                if (stp[i] == 0) { T[i] = kInf; inc[i] = (TT)0; continue; }
                const long long plane = (long long)(cur[i] + (stp[i] > 0 ? 1 : 0)) * kPsFix;
                T[i] = (TT)((plane - s[i]) * stp[i] * W[i]);
                inc[i] = (TT)((long long)kPsFix * W[i]);
            }
            // Every piece has positive length: T_i > 0 at the start (a source on a boundary belongs to the cell the ray
            // moves into) and all axes that reach Tn step together, so the next Tn is larger.  tau is summed in units
            // of T and scaled once.
            double tauT = 0.0;
            TT T0 = (TT)0;
            double r_in = 0.0, r_out = 0.0, dr = 0.0;
            // kappa of cell idx in the packed native copy: float index 2 o - (o & 1) if pair-packed, else 2 o
            // (rt_internal.h field_index; the bin offset is even).  The gather is software-pipelined: the kappa of the
            // cell a step moves into is requested as soon as that cell is known and used one step later, so that its
            // latency (L1 hit rate 78 %, the rest from L2) is covered by the step's own arithmetic instead of waited for
            // (long-scoreboard stalls were 5.3 warps per issue slot).
            // Two steps per loop turn with the two kappa registers swapping roles: a register move at the end of a
            // step would wait for the load it copies (it did: 29 % of all stall samples on that one move).
#define RT_PS_STEP(KUSE, KLOAD)                                                                                         \
            {                                                                                                           \
                const TT Tn = ps_min(T[0], ps_min(T[1], T[2]));                                                         \
                if (idx == idx_t) {                                 /* (padded linear indices of distinct cells differ) */ \
                    if (Tn == kInf) { r_in = 0.0; dr = r_out = 0.5 * (double)cell_width; }   /* source at this cell's centre */ \
                    else { r_in = (double)T0 * scale; dr = (double)(Tn - T0) * scale; r_out = r_in + dr; }              \
                    if (COUNT) nstep += 1;                                                                              \
                    break;                                                                                              \
                }                                                                                                       \
                const double dT = (double)(Tn - T0);                                                                    \
                if (COUNT) nstep += 1;                                                                                           \
                ps_advance(T[0], idx, Tn, inc[0], didx[0]);                                                             \
                ps_advance(T[1], idx, Tn, inc[1], didx[1]);                                                             \
                ps_advance(T[2], idx, Tn, inc[2], didx[2]);                                                             \
                KLOAD = fbin[2 * idx - (idx & ppN)];                /* the cell just entered (at the latest the target cell) */ \
                tauT = fma((double)KUSE, dT, tauT);                                                                     \
                T0 = Tn;                                                                                                \
            }
            float kap0 = fbin[2 * idx - (idx & ppN)], kap1 = 0.0f;
            for (;;) {
                RT_PS_STEP(kap0, kap1)
                RT_PS_STEP(kap1, kap0)
            }
#undef RT_PS_STEP
            const double tau = tauT * scale;
            const double dtau = (double)kap_t * dr;
            const double vol = 4.0 * 3.14159265358979323846 / 3.0 * dr * (r_out * r_out + r_out * r_in + r_in * r_in);
            q += (double)lum[(size_t)a * nbins + bin] * exp(-tau) * (-expm1(-dtau)) / vol;
            if (tau_out && a == diag_src && bin == diag_bin) tau_out[cidx] = (float)tau;
        }
        Q[(size_t)bin * ncell + cidx] = (float)q;
    }
    if (COUNT && steps && bin == 0) {
        unsigned n = nstep;
        for (int o = 16; o > 0; o >>= 1) n += __shfl_xor_sync(0xffffffffu, n, o);
        if ((threadIdx.x & 31) == 0 && n) atomicAdd(steps, (unsigned long long)n);
    }
}

cudaError_t launch_point_sources(float *Q, float *tau_out, const float2 *Pnat, int ppN, int nx, int ny, int nz, int nxp,
                                 const int *src_dev, const float *lum_dev, int nsrc, int nbins, int nbp, float cell_width,
                                 int diag_src, int diag_bin, unsigned long long *steps_dev, cudaStream_t st)
{
    const long long ncell = (long long)nx * ny * nz;
    dim3 grid((unsigned)((ncell + 127) / 128), 1, nbins);
    const bool small = nx <= 512 && ny <= 512 && nz <= 512, count = steps_dev != nullptr;
#define RT_PS_LAUNCH(TT, PP, COUNT)                                                                                      \
    k_point_sources<TT, PP, COUNT><<<grid, 128, 0, st>>>(Q, tau_out, Pnat, ppN, nx, ny, nz, nxp, src_dev, lum_dev, nsrc, nbins, nbp, \
                                                         cell_width, diag_src, diag_bin, steps_dev)
    if (small) {
        if (ppN) { if (count) RT_PS_LAUNCH(double, 1, true); else RT_PS_LAUNCH(double, 1, false); }
        else     { if (count) RT_PS_LAUNCH(double, 0, true); else RT_PS_LAUNCH(double, 0, false); }
    } else {
        if (ppN) { if (count) RT_PS_LAUNCH(long long, 1, true); else RT_PS_LAUNCH(long long, 1, false); }
        else     { if (count) RT_PS_LAUNCH(long long, 0, true); else RT_PS_LAUNCH(long long, 0, false); }
    }
#undef RT_PS_LAUNCH
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// Per-species rates of the point-source absorption (Appendix 1, eqs. A4-A6): one thread
// per cell, species and bins looped inside (elementwise; every array is read once, coalesced).
//   Gamma_i = (1/n_i) sum_b (kappa_ib / kappa_b) Q_b wG[i][b],  wG = 1 / h nu_b            for h nu_b >= h nu_i, else 0
//   Heat_i  = (1/n_i) sum_b (kappa_ib / kappa_b) Q_b wH[i][b],  wH = (h nu_b - h nu_i) / h nu_b
// ------------------------------------------------------------------------------------------------
__global__ void k_point_source_rates(float *__restrict__ Gamma, float *__restrict__ Heat, const float *__restrict__ Q,
                                     const float *__restrict__ ksp, const float *__restrict__ nsp,
                                     const float2 *__restrict__ Pnat, int ppN, int nx, int nxp, size_t rows, size_t ncell,
                                     int nbins, int nbp, int nspecies, const SpeciesWeights W)
{
    const float *__restrict__ fN = reinterpret_cast<const float *>(Pnat);
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < ncell; i += (size_t)gridDim.x * blockDim.x) {
        const size_t row = i / nx;
        const int x = (int)(i - row * nx);
        float g[kMaxSpecies], h[kMaxSpecies];
#pragma unroll
        for (int s = 0; s < kMaxSpecies; ++s) g[s] = h[s] = 0.0f;
        for (int b = 0; b < nbins; ++b) {
            const float kap = fN[field_index(packed_cell(b, row, x, nbp, nxp, rows), ppN)];
            const float qk = Q[(size_t)b * ncell + i] / kap;          // kappa > 0: floored in the packed copy
#pragma unroll
            for (int s = 0; s < kMaxSpecies; ++s)
                if (s < nspecies) {
                    const float part = ksp[((size_t)s * nbins + b) * ncell + i] * qk;      // (dtau_i / dtau) Q_b   (A4)
                    g[s] = fmaf(part, W.wG[s][b], g[s]);
                    h[s] = fmaf(part, W.wH[s][b], h[s]);
                }
        }
#pragma unroll
        for (int s = 0; s < kMaxSpecies; ++s)
            if (s < nspecies) {
                const float n = nsp[(size_t)s * ncell + i];
                Gamma[(size_t)s * ncell + i] = n > 0.0f ? g[s] / n : 0.0f;
                Heat[(size_t)s * ncell + i] = n > 0.0f ? h[s] / n : 0.0f;
            }
    }
}

cudaError_t launch_point_source_rates(float *Gamma, float *Heat, const float *Q, const float *ksp, const float *nsp,
                                      const float2 *Pnat, int ppN, int nx, int ny, int nz, int nxp, int nbins, int nbp,
                                      int nspecies, const SpeciesWeights &W, int sm_count, cudaStream_t st)
{
    const size_t ncell = (size_t)nx * ny * nz;
    size_t blocks = (ncell + 255) / 256;
    if (blocks > (size_t)sm_count * 8) blocks = (size_t)sm_count * 8;
    k_point_source_rates<<<(unsigned)blocks, 256, 0, st>>>(Gamma, Heat, Q, ksp, nsp, Pnat, ppN, nx, nxp, (size_t)ny * nz, ncell,
                                                           nbins, nbp, nspecies, W);
    return cudaGetLastError();
}

cudaError_t launch_counts_finalise(unsigned *counts, const float *accN, const float *accNC, int slotsN,
                                   const float *accT, const float *accTC, int slotsT,
                                   int nx, int ny, int nz, int nxp, int nyp, cudaStream_t st)
{
    for (long long zb0 = 0; zb0 < nz; zb0 += kMaxGridZ) {
        dim3 grid((nx + 31) / 32, (ny + 31) / 32, (unsigned)std::min<long long>(kMaxGridZ, nz - zb0)), block(32, 32);
        k_finalise<true><<<grid, block, 0, st>>>(nullptr, counts, nullptr, 0, accN, accNC, slotsN, accT, accTC, slotsT,
                                                 nx, ny, nz, nxp, nyp, 1, 1, 1.0f, 0, (int)zb0);
        const cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

__device__ __forceinline__ double warp_sum(double v)
{
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// out3 = {sum, min, max} over cells of (acc + accC); out3 must be pre-initialised to {0, +inf, 0}
__global__ void k_ds_reduce(double *out3, const float *__restrict__ acc, const float *__restrict__ accC, long long ncell,
                            int pitch, int width)
{
    double s = 0.0;
    float mn = 3.0e38f, mx = 0.0f;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < ncell; i += (long long)gridDim.x * blockDim.x) {
        if ((int)(i % pitch) >= width) continue;                 // pad cells of a row
        const float v = acc[i] + accC[i];
        s += (double)v;
        mn = fminf(mn, v); mx = fmaxf(mx, v);
    }
    s = warp_sum(s);
    for (int o = 16; o > 0; o >>= 1) {
        mn = fminf(mn, __shfl_xor_sync(0xffffffffu, mn, o));
        mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    }
    if ((threadIdx.x & 31) == 0) {
        atomicAdd(&out3[0], s);
        // non-negative doubles order like their bit patterns
        atomicMin(reinterpret_cast<unsigned long long *>(&out3[1]), (unsigned long long)__double_as_longlong((double)mn));
        atomicMax(reinterpret_cast<unsigned long long *>(&out3[2]), (unsigned long long)__double_as_longlong((double)mx));
    }
}

cudaError_t launch_ds_reduce(double *out3, const float *acc, const float *accC, long long ncell, int pitch, int width,
                             cudaStream_t st)
{
    int blocks = (int)((ncell + 1023) / 1024);
    if (blocks > 592) blocks = 592;
    k_ds_reduce<<<blocks, 256, 0, st>>>(out3, acc, accC, ncell, pitch, width);
    return cudaGetLastError();
}

// MODE_OWNERS: every element of w holds the number of stores it received in one launch (an exact small integer)
__global__ void k_owner_reduce(unsigned long long *out2, const float *__restrict__ w, long long n)
{
    unsigned mx = 0;
    unsigned long long s = 0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const unsigned v = __float2uint_rn(w[i]);
        mx = max(mx, v);
        s += v;
    }
    for (int o = 16; o > 0; o >>= 1) {
        mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, o));
        s += __shfl_xor_sync(0xffffffffu, s, o);
    }
    if ((threadIdx.x & 31) == 0) {
        atomicMax(&out2[0], (unsigned long long)mx);
        atomicAdd(&out2[1], s);
    }
}

cudaError_t launch_owner_reduce(unsigned long long *out2, const float *w, long long n, cudaStream_t st)
{
    int blocks = (int)((n + 1023) / 1024);
    if (blocks > 1184) blocks = 1184;
    k_owner_reduce<<<blocks, 256, 0, st>>>(out2, w, n);
    return cudaGetLastError();
}

__global__ void k_sum_u32(unsigned long long *out, const unsigned *__restrict__ c, long long n)
{
    unsigned long long s = 0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) s += c[i];
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) atomicAdd(out, s);
}

cudaError_t launch_sum_u32(unsigned long long *out, const unsigned *counts, long long n, cudaStream_t st)
{
    int blocks = (int)((n + 1023) / 1024);
    if (blocks > 592) blocks = 592;
    k_sum_u32<<<blocks, 256, 0, st>>>(out, counts, n);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// Streaming bandwidth probe (rt_probe_bandwidth): the roofline denominators of the memory levels that
// MEASURED_PEAKS.json does not carry (L2), measured with the same instruction mix the sweep's memory side has:
// 16-byte cache-global loads, and a read-modify-write of every element.
// ------------------------------------------------------------------------------------------------
template <int RMW>
__global__ void __launch_bounds__(512) k_probe(float4 *__restrict__ buf, size_t n4, int reps, float4 *__restrict__ sink)
{
    // `reps` passes over the buffer inside one launch (a single pass over an L2-sized buffer lasts a few microseconds,
    // less than a launch); four independent 16-byte accesses per thread and iteration
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int r = 0; r < reps; ++r) {
        size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
        for (; i + 3 * stride < n4; i += 4 * stride) {
            float4 v0 = __ldcg(buf + i), v1 = __ldcg(buf + i + stride), v2 = __ldcg(buf + i + 2 * stride), v3 = __ldcg(buf + i + 3 * stride);
            if (RMW) {
                v0.x += 1.0f; v1.x += 1.0f; v2.x += 1.0f; v3.x += 1.0f;
                __stcg(buf + i, v0); __stcg(buf + i + stride, v1); __stcg(buf + i + 2 * stride, v2); __stcg(buf + i + 3 * stride, v3);
            } else {
                acc.x += v0.x + v1.x + v2.x + v3.x; acc.y += v0.y + v1.y + v2.y + v3.y;
                acc.z += v0.z + v1.z + v2.z + v3.z; acc.w += v0.w + v1.w + v2.w + v3.w;
            }
        }
        for (; i < n4; i += stride) {
            float4 v = __ldcg(buf + i);
            if (RMW) { v.x += 1.0f; __stcg(buf + i, v); }
            else { acc.x += v.x; acc.y += v.y; acc.z += v.z; acc.w += v.w; }
        }
    }
    if (!RMW && acc.x + acc.y + acc.z + acc.w == -1.0f) *sink = acc;      // never true for the zeroed buffer: keeps the loads
}

cudaError_t launch_probe(float4 *buf, size_t n4, int rmw, int reps, int sm_count, cudaStream_t st)
{
    const int blocks = 8 * sm_count;
    if (rmw) k_probe<1><<<blocks, 512, 0, st>>>(buf, n4, reps, buf);
    else     k_probe<0><<<blocks, 512, 0, st>>>(buf, n4, reps, buf);
    return cudaGetLastError();
}

}  // namespace rt
