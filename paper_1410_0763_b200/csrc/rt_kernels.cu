// sm_100a kernels of the diffuse-radiation ray sweep (arXiv:1410.0763 section 2.2 / 3.1).
//
//   k_build_programs   integer traversal of one slab for all rays of a direction (Fig. 2)
//   k_pack_fields      (kappa, S) -> packed float2 copies: native [z][y][x] and transposed [x][z][y]
//   k_sweep_owned      the hot kernel: eq. 7 / eq. 8 per segment, atomic-free J partials by cell ownership
//   k_sweep_generic    one thread per lattice ray with per-ray integer traversal; the paper's four
//                      ray groups or atomicAdd -- ablations and fallback
//   k_normalise        eqs. 10-13: sum slot/seam accumulators, 1/(N_d kappa), + S
//   diagnostics        counts finalise, sum-of-ds reduction
//
// See DESIGN.md for the data layout and why the ownership scheme replaces the four ray groups.
#include "rt_internal.h"

namespace rt {

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
    // fractional entry position inside the entry cell; the same for every lattice ray (offsets are
    // whole cells): U = p*ONE + ONE/2 + k*Mb
    const long long u = (ONE / 2 + (long long)k * Mb) & (ONE - 1);
    const long long v = (ONE / 2 + (long long)k * Mc) & (ONE - 1);
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
    s.len0 = (float)(l0 * Lw); s.len1 = (float)(l1 * Lw); s.len2 = (float)(l2 * Lw); s.flags = f;
    prog[D.prog_off + k] = s;
}

cudaError_t launch_build_programs(const DirDev *dirs, int ndirs, SlabProg *prog, double cell_width,
                                  const double *Lvals, cudaStream_t st)
{
    // Na <= max dim; launch enough threads for the largest (bounded by 65535 blocks in y: loop)
    int maxNa = 1 << 16;   // generous upper bound handled by the k >= Na guard
    (void)maxNa;
    for (int d0 = 0; d0 < ndirs; d0 += 32768) {
        int nd = ndirs - d0 < 32768 ? ndirs - d0 : 32768;
        dim3 grid(64, nd);     // 64*256 = 16384 slabs max
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
                              float2 *__restrict__ Pnat, float2 *__restrict__ PT, int nx, int ny, int nz)
{
    __shared__ float2 tile[32][33];
    const int bin = blockIdx.z / nz, z = blockIdx.z % nz;
    const int x0 = blockIdx.x * 32, y0 = blockIdx.y * 32;
    const size_t ncell = (size_t)nx * ny * nz;
    const size_t boff = (size_t)bin * ncell;
    for (int dy = threadIdx.y; dy < 32; dy += blockDim.y) {
        int x = x0 + threadIdx.x, y = y0 + dy;
        if (x < nx && y < ny) {
            size_t i = boff + ((size_t)z * ny + y) * nx + x;
            float2 v = make_float2(fmaxf(kappa[i], kKappaMin), S[i]);
            Pnat[i] = v;
            tile[dy][threadIdx.x] = v;
        }
    }
    __syncthreads();
    for (int dx = threadIdx.y; dx < 32; dx += blockDim.y) {
        int x = x0 + dx, y = y0 + threadIdx.x;
        if (x < nx && y < ny)
            PT[boff + ((size_t)x * nz + z) * ny + y] = tile[threadIdx.x][dx];
    }
}

cudaError_t launch_pack_fields(const float *kappa, const float *S, float2 *Pnat, float2 *PT,
                               int nx, int ny, int nz, int nbins, cudaStream_t st)
{
    dim3 grid((nx + 31) / 32, (ny + 31) / 32, nz * nbins), block(32, 8);
    k_pack_fields<<<grid, block, 0, st>>>(kappa, S, Pnat, PT, nx, ny, nz);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// Segment update (eq. 7, eq. 8), fp32
//   A = 1 - exp(-kappa*len); contribution to the cell += I_in * A  (numerator of eq. 11 times kappa*L,
//   see DESIGN.md "Arithmetic"); I_out = I_in * e + S * A with e = exp(-kappa*len).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ float ex2_approx(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// e = exp(-kappa*len) and A = 1 - e, each with small RELATIVE error: e straight from ex2 (never as
// 1 - A: behind an opaque cell the transmitted part I*e is all that is left), A from a polynomial
// where 1 - e would cancel.
__device__ __forceinline__ float one_minus_exp(float kap, float len, float ct, float &e)
{
    const float x = kap * len;
    e = ex2_approx(kap * ct);                                  // ct = -len*log2(e)
    // small-x branch: x * (c0 + c1 x + c2 x^2 + c3 x^3), fitted on [0, 1/4]; rel. error 3.4e-7
    float p = fmaf(x, -0.0377338513f, 0.1660640817f);
    p = fmaf(x, p, -0.4999701648f);
    p = fmaf(x, p, 0.9999997683f);
    return x < 0.25f ? x * p : 1.0f - e;
}

template <int MODE>
__device__ __forceinline__ void seg_update(float &I, float kap, float src, float len, float ct, float &part)
{
    if (MODE == MODE_J) {
        float e;
        const float A = one_minus_exp(kap, len, ct, e);
        part = fmaf(I, A, part);
        I = fmaf(I, e, src * A);                               // eq. 7
    } else if (MODE == MODE_COUNT) {
        part += 1.0f;
    } else {
        part += len;
    }
}

// ------------------------------------------------------------------------------------------------
// The owned sweep kernel.
//
// One warp owns R consecutive rays rows (transverse axis c) over the full cyclic extent of the
// memory-contiguous transverse axis b: Nb = 32*CW*G columns, each thread owning G chunks of CW
// adjacent columns (aligned vector loads).  Along b the thread owns CELLS: a ray that crosses a
// b-boundary is handed to the owner of the next column (register move / one rotate shuffle per
// chunk; a chunk-to-chunk carry; leaving the last column = leaving the box, and a new ray with the
// inflow intensity enters the first column).  Along c the warp owns RAYS: the memory row of ray
// row r is (q0 + r + shift_k) mod Nc, pure address arithmetic; pieces that fall into the next
// memory row use the next row's data and add to the next row's partial, both held by the same
// thread.  Only the partial of the row above the warp's last ray row has another owner; it goes
// to the seam accumulator accC with plain stores.  Every cell therefore has exactly one writer
// per accumulator array and launch: no atomics, deterministic sums.
// ------------------------------------------------------------------------------------------------
template <int CW> struct VecT;
template <> struct VecT<2> { using D = float4; using A = float2; };
template <> struct VecT<1> { using D = float2; using A = float;  };

template <int CW>
__device__ __forceinline__ void unpack(const typename VecT<CW>::D &v, float (&kap)[CW], float (&src)[CW]);
template <>
__device__ __forceinline__ void unpack<2>(const float4 &v, float (&kap)[2], float (&src)[2])
{ kap[0] = v.x; src[0] = v.y; kap[1] = v.z; src[1] = v.w; }
template <>
__device__ __forceinline__ void unpack<1>(const float2 &v, float (&kap)[1], float (&src)[1])
{ kap[0] = v.x; src[0] = v.y; }

constexpr int kWarpsPerCta = 4;

template <int CW>
__device__ __forceinline__ typename VecT<CW>::A acc_new(const typename VecT<CW>::A &o, const float (&part)[CW], float w);
template <>
__device__ __forceinline__ float2 acc_new<2>(const float2 &o, const float (&part)[2], float w)
{ return make_float2(fmaf(part[0], w, o.x), fmaf(part[1], w, o.y)); }
template <>
__device__ __forceinline__ float acc_new<1>(const float &o, const float (&part)[1], float w)
{ return fmaf(part[0], w, o); }

// The six slab patterns that occur away from exact boundary touches get straight-line code
// (FLC = compile-time flags); anything else runs the same body with run-time flags (FLC < 0).
constexpr int kPatNone = 0;
constexpr int kPatB    = F_SB1 | F_P1;
constexpr int kPatC    = F_SC1 | F_P1;
constexpr int kPatBC   = F_SB1 | F_P1 | F_SC2 | F_P2;
constexpr int kPatCB   = F_SC1 | F_P1 | F_SB2 | F_P2;
constexpr int kPatD    = F_SB1 | F_SC1 | F_P1;

// One slab for the R rays rows of a warp.  `src` supplies the slab's inputs: data(r, g) = packed
// (kappa, S) of chunk g of memory row (lbase + r) (r = R: the seam row, valid only if some piece
// steps along c), acc(r, g) / accC(g) = old accumulator values of the rows this warp owns / of
// the seam row.  New accumulator values go straight to global memory (one writer per cell).
template <int CW, int G, int R, int MODE, int FLC, class Src>
__device__ __forceinline__ void slab_rows(const unsigned fl_rt, float (&I)[R][G][CW], const Src &src,
                                          const float len0, const float len1, const float len2,
                                          const float Ibc, const float invL, const int lane, const bool rev,
                                          const int lbase, const int Nc,
                                          float *__restrict__ acc, float *__restrict__ accC,
                                          const long long (&orow)[R + 1], const int (&col)[G])
{
    using AV = typename VecT<CW>::A;
    constexpr unsigned FULL = 0xffffffffu;
    constexpr float LOG2E = 1.4426950408889634f;
    const unsigned fl = (FLC >= 0) ? (unsigned)FLC : fl_rt;
    const float ct0 = -len0 * LOG2E, ct1 = -len1 * LOG2E, ct2 = -len2 * LOG2E;
    const bool anySC = (fl & (F_SC1 | F_SC2)) != 0;

    float part_cur[G][CW];
#pragma unroll
    for (int g = 0; g < G; ++g)
#pragma unroll
        for (int i = 0; i < CW; ++i) part_cur[g][i] = 0.0f;

#pragma unroll
    for (int r = 0; r < R; ++r) {
        int l_r = lbase + r; if (l_r >= Nc) l_r -= Nc;
        const bool wrap_r = (l_r == Nc - 1);
        float part_next[G][CW];
#pragma unroll
        for (int g = 0; g < G; ++g)
#pragma unroll
            for (int i = 0; i < CW; ++i) part_next[g][i] = 0.0f;

        float carry = Ibc;            // intensity handed from chunk g-1 (a new ray for g = 0)
#pragma unroll
        for (int g = 0; g < G; ++g) {
            float kc[CW], sc[CW], kn[CW], sn[CW];
            unpack<CW>(src.data(r, g), kc, sc);
            if (anySC) unpack<CW>(src.data(r + 1, g), kn, sn);
            else { 
#pragma unroll
                for (int i = 0; i < CW; ++i) { kn[i] = kc[i]; sn[i] = sc[i]; }
            }
            float (&Iu)[CW] = I[r][g];
#pragma unroll
            for (int i = 0; i < CW; ++i) seg_update<MODE>(Iu[i], kc[i], sc[i], len0, ct0, part_cur[g][i]);
            bool sel = false;
#pragma unroll
            for (int stage = 1; stage <= 2; ++stage) {
                const unsigned fsb = (stage == 1) ? F_SB1 : F_SB2;
                const unsigned fsc = (stage == 1) ? F_SC1 : F_SC2;
                const unsigned fp = (stage == 1) ? F_P1 : F_P2;
                const float len = (stage == 1) ? len1 : len2;
                const float ct = (stage == 1) ? ct1 : ct2;
                if (fl & (fsb | fsc)) {
                    if (MODE == MODE_J) {
                        if (fl & fsb) {       // step along b: hand every ray to the next column's owner
                            const float out = rev ? Iu[0] : Iu[CW - 1];
                            const float t = __shfl_sync(FULL, out, (lane + 31) & 31);
                            const float in = (lane == 0) ? carry : t;
                            carry = t;
                            if (CW == 2) {
                                const float keep = rev ? Iu[CW - 1] : Iu[0];
                                Iu[0] = rev ? keep : in;
                                Iu[CW - 1] = rev ? in : keep;
                            } else {
                                Iu[0] = in;
                            }
                        }
                        if ((fl & fsc) && wrap_r) {   // step along c out of the box: new rays enter
#pragma unroll
                            for (int i = 0; i < CW; ++i) Iu[i] = Ibc;
                        }
                    }
                    if (fl & fsc) sel = true;
                }
                if (fl & fp) {
                    if (sel) {
#pragma unroll
                        for (int i = 0; i < CW; ++i) seg_update<MODE>(Iu[i], kn[i], sn[i], len, ct, part_next[g][i]);
                    } else {
#pragma unroll
                        for (int i = 0; i < CW; ++i) seg_update<MODE>(Iu[i], kc[i], sc[i], len, ct, part_cur[g][i]);
                    }
                }
            }
        }
        // row r's partial is complete (own pieces + pieces of ray row r-1 that stepped along c)
#pragma unroll
        for (int g = 0; g < G; ++g)
            *reinterpret_cast<AV *>(acc + orow[r] + col[g]) = acc_new<CW>(src.acc(r, g), part_cur[g], invL);
#pragma unroll
        for (int g = 0; g < G; ++g)
#pragma unroll
            for (int i = 0; i < CW; ++i) part_cur[g][i] = part_next[g][i];
    }
    if (anySC) {
        // seam: the partial of the memory row above the warp's last ray row has another owner
#pragma unroll
        for (int g = 0; g < G; ++g)
            *reinterpret_cast<AV *>(accC + orow[R] + col[g]) = acc_new<CW>(src.accC(g), part_cur[g], invL);
    }
}

// ---- mirror pairs ---------------------------------------------------------------------------------
// Two directions that differ only by the sign of their component along the memory-contiguous
// transverse axis b (HEALPix sets are symmetric under x -> -x and y -> -y) have the
// same slab programs, the same row drift along c and the same dominant-axis march: at every slab a
// warp that carries both touches the SAME cells with the SAME piece lengths.  So the packed field
// rows and the accumulator rows are moved once for the two directions, and e = exp(-kappa ds),
// A = 1 - e and S*A are evaluated once per (cell, piece) and applied to both intensities.  Only
// the b-step differs: rays of direction 0 are handed to the next higher column, rays of direction
// 1 to the next lower one.  Stage-major order (all chunks do piece 0, then the step, ...) because
// the two directions need their chunk-to-chunk carries in opposite chunk order.
template <int MODE>
__device__ __forceinline__ void seg_update2(float &I0, float &I1, float kap, float src, float len, float ct, float &part)
{
    if (MODE == MODE_J) {
        float e;
        const float A = one_minus_exp(kap, len, ct, e);
        const float SA = src * A;
        part = fmaf(I0 + I1, A, part);
        I0 = fmaf(I0, e, SA);                                  // eq. 7, direction 0
        I1 = fmaf(I1, e, SA);                                  // eq. 7, mirrored direction
    } else if (MODE == MODE_COUNT) {
        part += 2.0f;
    } else {
        part += 2.0f * len;
    }
}

template <int CW, int G, int R, int MODE, int FLC, class Src>
__device__ __forceinline__ void slab_rows_pair(const unsigned fl_rt, float (&I)[2][R][G][CW], const Src &src,
                                               const float len0, const float len1, const float len2,
                                               const float Ibc, const float invL, const int lane,
                                               const int lbase, const int Nc,
                                               float *__restrict__ acc, float *__restrict__ accC,
                                               const long long (&orow)[R + 1], const int (&col)[G])
{
    using AV = typename VecT<CW>::A;
    constexpr unsigned FULL = 0xffffffffu;
    constexpr float LOG2E = 1.4426950408889634f;
    const unsigned fl = (FLC >= 0) ? (unsigned)FLC : fl_rt;
    const float ct0 = -len0 * LOG2E, ct1 = -len1 * LOG2E, ct2 = -len2 * LOG2E;
    const bool anySC = (fl & (F_SC1 | F_SC2)) != 0;

    float part_cur[G][CW];
#pragma unroll
    for (int g = 0; g < G; ++g)
#pragma unroll
        for (int i = 0; i < CW; ++i) part_cur[g][i] = 0.0f;

#pragma unroll
    for (int r = 0; r < R; ++r) {
        int l_r = lbase + r; if (l_r >= Nc) l_r -= Nc;
        const bool wrap_r = (l_r == Nc - 1);
        float part_next[G][CW];
        float kc[G][CW], sc[G][CW], kn[G][CW], sn[G][CW];
#pragma unroll
        for (int g = 0; g < G; ++g) {
            unpack<CW>(src.data(r, g), kc[g], sc[g]);
            if (anySC) unpack<CW>(src.data(r + 1, g), kn[g], sn[g]);
#pragma unroll
            for (int i = 0; i < CW; ++i) {
                part_next[g][i] = 0.0f;
                if (!anySC) { kn[g][i] = kc[g][i]; sn[g][i] = sc[g][i]; }
            }
        }
        float (&I0)[G][CW] = I[0][r];
        float (&I1)[G][CW] = I[1][r];
#pragma unroll
        for (int g = 0; g < G; ++g)
#pragma unroll
            for (int i = 0; i < CW; ++i) seg_update2<MODE>(I0[g][i], I1[g][i], kc[g][i], sc[g][i], len0, ct0, part_cur[g][i]);
        bool sel = false;
#pragma unroll
        for (int stage = 1; stage <= 2; ++stage) {
            const unsigned fsb = (stage == 1) ? F_SB1 : F_SB2;
            const unsigned fsc = (stage == 1) ? F_SC1 : F_SC2;
            const unsigned fp = (stage == 1) ? F_P1 : F_P2;
            const float len = (stage == 1) ? len1 : len2;
            const float ct = (stage == 1) ? ct1 : ct2;
            if (fl & (fsb | fsc)) {
                if (MODE == MODE_J) {
                    if (fl & fsb) {
                        // direction 0: every ray to the next higher column; a new ray enters column 0
                        float carry = Ibc;
#pragma unroll
                        for (int g = 0; g < G; ++g) {
                            const float t = __shfl_sync(FULL, I0[g][CW - 1], (lane + 31) & 31);
                            const float in = (lane == 0) ? carry : t;
                            carry = t;
                            if (CW == 2) I0[g][CW - 1] = I0[g][0];
                            I0[g][0] = in;
                        }
                        // direction 1: every ray to the next lower column; a new ray enters the last column
                        carry = Ibc;
#pragma unroll
                        for (int g = G - 1; g >= 0; --g) {
                            const float t = __shfl_sync(FULL, I1[g][0], (lane + 1) & 31);
                            const float in = (lane == 31) ? carry : t;
                            carry = t;
                            if (CW == 2) I1[g][0] = I1[g][CW - 1];
                            I1[g][CW - 1] = in;
                        }
                    }
                    if ((fl & fsc) && wrap_r) {   // step along c out of the box: new rays enter
#pragma unroll
                        for (int g = 0; g < G; ++g)
#pragma unroll
                            for (int i = 0; i < CW; ++i) { I0[g][i] = Ibc; I1[g][i] = Ibc; }
                    }
                }
                if (fl & fsc) sel = true;
            }
            if (fl & fp) {
#pragma unroll
                for (int g = 0; g < G; ++g)
#pragma unroll
                    for (int i = 0; i < CW; ++i) {
                        if (sel) seg_update2<MODE>(I0[g][i], I1[g][i], kn[g][i], sn[g][i], len, ct, part_next[g][i]);
                        else     seg_update2<MODE>(I0[g][i], I1[g][i], kc[g][i], sc[g][i], len, ct, part_cur[g][i]);
                    }
            }
        }
#pragma unroll
        for (int g = 0; g < G; ++g)
            *reinterpret_cast<AV *>(acc + orow[r] + col[g]) = acc_new<CW>(src.acc(r, g), part_cur[g], invL);
#pragma unroll
        for (int g = 0; g < G; ++g)
#pragma unroll
            for (int i = 0; i < CW; ++i) part_cur[g][i] = part_next[g][i];
    }
    if (anySC) {
#pragma unroll
        for (int g = 0; g < G; ++g)
            *reinterpret_cast<AV *>(accC + orow[R] + col[g]) = acc_new<CW>(src.accC(g), part_cur[g], invL);
    }
}

#define RT_DISPATCH_SLAB_PAIR(fl, ...)                                                    \
    switch (fl) {                                                                         \
    case kPatNone: slab_rows_pair<CW, G, R, MODE, kPatNone>(__VA_ARGS__); break;          \
    case kPatB:    slab_rows_pair<CW, G, R, MODE, kPatB>(__VA_ARGS__); break;             \
    case kPatC:    slab_rows_pair<CW, G, R, MODE, kPatC>(__VA_ARGS__); break;             \
    case kPatBC:   slab_rows_pair<CW, G, R, MODE, kPatBC>(__VA_ARGS__); break;            \
    case kPatCB:   slab_rows_pair<CW, G, R, MODE, kPatCB>(__VA_ARGS__); break;            \
    case kPatD:    slab_rows_pair<CW, G, R, MODE, kPatD>(__VA_ARGS__); break;             \
    default:       slab_rows_pair<CW, G, R, MODE, -1>(__VA_ARGS__); break;                \
    }

#define RT_DISPATCH_SLAB(fl, ...)                                                         \
    switch (fl) {                                                                         \
    case kPatNone: slab_rows<CW, G, R, MODE, kPatNone>(__VA_ARGS__); break;               \
    case kPatB:    slab_rows<CW, G, R, MODE, kPatB>(__VA_ARGS__); break;                  \
    case kPatC:    slab_rows<CW, G, R, MODE, kPatC>(__VA_ARGS__); break;                  \
    case kPatBC:   slab_rows<CW, G, R, MODE, kPatBC>(__VA_ARGS__); break;                 \
    case kPatCB:   slab_rows<CW, G, R, MODE, kPatCB>(__VA_ARGS__); break;                 \
    case kPatD:    slab_rows<CW, G, R, MODE, kPatD>(__VA_ARGS__); break;                  \
    default:       slab_rows<CW, G, R, MODE, -1>(__VA_ARGS__); break;                     \
    }

// row shift of slab k in closed form: floor(1/2 + k m_c), m_c in units of 2^-20
__device__ __forceinline__ int row_shift(int k, int Mc) { return (int)(((kOne >> 1) + (long long)k * Mc) >> kF); }

// ---- variant A: inputs loaded straight into registers at the top of each slab ----------------------
template <int CW, int G, int R>
struct RegSrc {
    using DV = typename VecT<CW>::D;
    using AV = typename VecT<CW>::A;
    DV rowd[R + 1][G];
    AV acco[R][G], accCo[G];
    __device__ __forceinline__ const DV &data(int r, int g) const { return rowd[r][g]; }
    __device__ __forceinline__ const AV &acc(int r, int g) const { return acco[r][g]; }
    __device__ __forceinline__ const AV &accC(int g) const { return accCo[g]; }
};

template <int CW, int G, int R, int MODE>
__global__ void __launch_bounds__(32 * kWarpsPerCta)
k_sweep_owned(const SweepLaunch L)
{
    using DV = typename VecT<CW>::D;
    using AV = typename VecT<CW>::A;

    const int lane = threadIdx.x & 31;
    const int slot = blockIdx.y, bin = blockIdx.z;
    const DirDev *__restrict__ Dp = L.dirs + L.batch[slot];
    const int Nc = Dp->Nc, Na = Dp->Na, Mc = Dp->Mc;
    const int q0 = (blockIdx.x * kWarpsPerCta + (threadIdx.x >> 5)) * R;
    if (q0 >= Nc) return;
    const long long sk = Dp->sk, sl = Dp->sl;
    const bool rev = Dp->sj < 0;
    const float invL = (MODE == MODE_J) ? Dp->invL : 1.0f;
    const float Ibc = L.Ibc[bin];
    const SlabProg *__restrict__ prog = L.prog + Dp->prog_off;

    const long long foff = (long long)bin * L.ncell + Dp->base;
    const float2 *__restrict__ P = L.P + foff;
    float *__restrict__ acc = L.acc + ((long long)slot * L.nbins) * L.ncell + foff;
    float *__restrict__ accC = L.accC + ((long long)slot * L.nbins) * L.ncell + foff;

    // canonical chunk g / lane -> first memory column of the chunk (rays move +1 in canonical order)
    int col[G];
#pragma unroll
    for (int g = 0; g < G; ++g)
        col[g] = rev ? (32 * CW * G - CW * (32 * g + lane + 1)) : CW * (32 * g + lane);

    float I[R][G][CW];
#pragma unroll
    for (int r = 0; r < R; ++r)
#pragma unroll
        for (int g = 0; g < G; ++g)
#pragma unroll
            for (int i = 0; i < CW; ++i) I[r][g][i] = Ibc;

    RegSrc<CW, G, R> src;
    long long orow[R + 1];
    SlabProg pr = prog[0];

    for (int k = 0; k < Na; ++k) {
        const unsigned fl = pr.flags;
        const float len0 = pr.len0, len1 = pr.len1, len2 = pr.len2;
        if (k + 1 < Na) pr = prog[k + 1];
        const int lbase = (q0 + row_shift(k, Mc)) % Nc;
        const long long offk = (long long)k * sk;
#pragma unroll
        for (int r = 0; r <= R; ++r) {
            int l = lbase + r; if (l >= Nc) l -= Nc;
            orow[r] = offk + (long long)l * sl;
        }
#pragma unroll
        for (int r = 0; r < R; ++r)
#pragma unroll
            for (int g = 0; g < G; ++g) {
                src.rowd[r][g] = *reinterpret_cast<const DV *>(P + orow[r] + col[g]);
                src.acco[r][g] = *reinterpret_cast<const AV *>(acc + orow[r] + col[g]);
            }
        if (fl & (F_SC1 | F_SC2)) {
#pragma unroll
            for (int g = 0; g < G; ++g) {
                src.rowd[R][g] = *reinterpret_cast<const DV *>(P + orow[R] + col[g]);
                src.accCo[g] = *reinterpret_cast<const AV *>(accC + orow[R] + col[g]);
            }
        }
        RT_DISPATCH_SLAB(fl, fl, I, src, len0, len1, len2, Ibc, invL, lane, rev, lbase, Nc, acc, accC, orow, col)
    }
}

// ---- variant B: inputs staged in a warp-private shared-memory ring by the TMA engine ---------------
// Each warp owns D stages; stage (k mod D) holds slab k's packed field rows and old accumulator
// rows, copied by 1-D bulk async copies (cp.async.bulk, SASS UBLKCP) issued by lane 0 D slabs ahead
// and tracked by one mbarrier per stage (transaction-byte count).  No registers are spent on data in
// flight, so the prefetch depth is set by shared memory, not by the register file.
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count)
{ asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(bar), "r"(count) : "memory"); }
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes)
{ asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(bar), "r"(bytes) : "memory"); }
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@!p bra WAIT_%=;\n\t}"
        :: "r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(unsigned dst, const void *src, unsigned bytes, unsigned bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 :: "r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}

template <int CW, int G, int R>
struct SmemSrc {
    using DV = typename VecT<CW>::D;
    using AV = typename VecT<CW>::A;
    static constexpr int kNb = 32 * CW * G;
    static constexpr int kRowP = kNb * (int)sizeof(float2);
    static constexpr int kRowA = kNb * (int)sizeof(float);
    static constexpr int kStage = (R + 1) * (kRowP + kRowA);
    const unsigned char *stage;      // generic pointer to the stage in shared memory
    int colb;                        // byte offset of this lane's chunk 0 within a float2 row (fwd) ...
    int cstep;                       // ... and signed chunk stride in float2 elements
    int col0;                        // first column of chunk 0
    __device__ __forceinline__ DV data(int r, int g) const
    { return *reinterpret_cast<const DV *>(stage + r * kRowP + (col0 + g * cstep) * (int)sizeof(float2)); }
    __device__ __forceinline__ AV acc(int r, int g) const
    { return *reinterpret_cast<const AV *>(stage + (R + 1) * kRowP + r * kRowA + (col0 + g * cstep) * (int)sizeof(float)); }
    __device__ __forceinline__ AV accC(int g) const { return acc(R, g); }
};

template <int CW, int G, int R, int MODE, int D, int ND>
__global__ void __launch_bounds__(32 * kWarpsPerCta)
k_sweep_tma(const SweepLaunch L)
{
    using Src = SmemSrc<CW, G, R>;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    constexpr int kWarpBytes = D * Src::kStage + 128;

    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int slot = blockIdx.y, bin = blockIdx.z;
    const DirDev *__restrict__ Dp = L.dirs + L.batch[slot];
    const int Nc = Dp->Nc, Na = Dp->Na, Mc = Dp->Mc;
    const int q0 = (blockIdx.x * kWarpsPerCta + wid) * R;
    if (q0 >= Nc) return;
    const long long sk = Dp->sk, sl = Dp->sl;
    const bool rev = Dp->sj < 0;
    const float invL = (MODE == MODE_J) ? Dp->invL : 1.0f;
    const float Ibc = L.Ibc[bin];
    const SlabProg *__restrict__ prog = L.prog + Dp->prog_off;

    const long long foff = (long long)bin * L.ncell + Dp->base;
    const float2 *__restrict__ P = L.P + foff;
    float *__restrict__ acc = L.acc + ((long long)slot * L.nbins) * L.ncell + foff;
    float *__restrict__ accC = L.accC + ((long long)slot * L.nbins) * L.ncell + foff;

    unsigned char *wbase = smem_raw + wid * kWarpBytes;
    const unsigned wbase_s = smem_u32(wbase);
    const unsigned bars = wbase_s + D * Src::kStage;
    if (lane == 0) {
#pragma unroll
        for (int s = 0; s < D; ++s) mbar_init(bars + 8 * s, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncwarp();

    int col[G];
#pragma unroll
    for (int g = 0; g < G; ++g)
        col[g] = rev ? (32 * CW * G - CW * (32 * g + lane + 1)) : CW * (32 * g + lane);

    // producer: lane 0 asks the TMA engine for slab kk's rows
    auto produce = [&](int kk) {
        if (lane != 0) return;
        const int s = kk % D;
        const unsigned st = wbase_s + s * Src::kStage, bar = bars + 8 * s;
        const int s0 = row_shift(kk, Mc), s1 = row_shift(kk + 1, Mc);
        const bool seam = (s1 != s0);
        const int lb = (q0 + s0) % Nc;
        const long long offk = (long long)kk * sk;
        const int nrows = R + (seam ? 1 : 0);
        mbar_expect_tx(bar, (unsigned)(nrows * ((MODE == MODE_J ? Src::kRowP : 0) + Src::kRowA)));
#pragma unroll
        for (int r = 0; r <= R; ++r) {
            if (r == R && !seam) break;
            int l = lb + r; if (l >= Nc) l -= Nc;
            const long long o = offk + (long long)l * sl;
            if (MODE == MODE_J) bulk_g2s(st + r * Src::kRowP, P + o, Src::kRowP, bar);
            bulk_g2s(st + (R + 1) * Src::kRowP + r * Src::kRowA, (r < R ? acc : accC) + o, Src::kRowA, bar);
        }
    };
#pragma unroll 1
    for (int kk = 0; kk < D && kk < Na; ++kk) produce(kk);

    float I[ND][R][G][CW];
#pragma unroll
    for (int d = 0; d < ND; ++d)
#pragma unroll
        for (int r = 0; r < R; ++r)
#pragma unroll
            for (int g = 0; g < G; ++g)
#pragma unroll
                for (int i = 0; i < CW; ++i) I[d][r][g][i] = Ibc;

    Src src;
    src.col0 = col[0];
    src.cstep = rev ? -32 * CW : 32 * CW;
    src.colb = 0;
    long long orow[R + 1];
    SlabProg pr = prog[0];

#pragma unroll 1
    for (int k = 0; k < Na; ++k) {
        const unsigned fl = pr.flags;
        const float len0 = pr.len0, len1 = pr.len1, len2 = pr.len2;
        if (k + 1 < Na) pr = prog[k + 1];
        const int lbase = (q0 + row_shift(k, Mc)) % Nc;
        const long long offk = (long long)k * sk;
#pragma unroll
        for (int r = 0; r <= R; ++r) {
            int l = lbase + r; if (l >= Nc) l -= Nc;
            orow[r] = offk + (long long)l * sl;
        }
        const int s = k % D;
        src.stage = wbase + s * Src::kStage;
        mbar_wait(bars + 8 * s, (unsigned)((k / D) & 1));
        if constexpr (ND == 2) {
            RT_DISPATCH_SLAB_PAIR(fl, fl, I, src, len0, len1, len2, Ibc, invL, lane, lbase, Nc, acc, accC, orow, col)
        } else {
            RT_DISPATCH_SLAB(fl, fl, I[0], src, len0, len1, len2, Ibc, invL, lane, rev, lbase, Nc, acc, accC, orow, col)
        }
        __syncwarp();                     // every lane is done reading stage s
        if (k + D < Na) produce(k + D);
    }
}

bool owned_supported(int Nb, int Nc, int rows)
{
    if (!(Nb == 32 || Nb == 64 || Nb == 128 || Nb == 256)) return false;
    if (!(rows == 1 || rows == 2 || rows == 4)) return false;
    return Nc % rows == 0;
}

template <int CW, int G, int R, int MODE>
static cudaError_t launch_owned_one(const SweepLaunch &L, cudaStream_t st)
{
    const int tiles = L.Nc / R;
    dim3 grid((tiles + kWarpsPerCta - 1) / kWarpsPerCta, L.nslots, L.nbins), block(32 * kWarpsPerCta);
    if (L.stages >= 2) {
        using Src = SmemSrc<CW, G, R>;
        auto go = [&](auto kern, int D) -> cudaError_t {
            const int smem = kWarpsPerCta * (D * Src::kStage + 128);
            if (smem > 227 * 1024) return cudaErrorInvalidValue;
            cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
            if (e != cudaSuccess) return e;
            kern<<<grid, block, smem, st>>>(L);
            return cudaGetLastError();
        };
        if constexpr (MODE == MODE_J) {
            if (L.pair) {
                switch (L.stages) {
                case 2: return go(k_sweep_tma<CW, G, R, MODE, 2, 2>, 2);
                case 3: return go(k_sweep_tma<CW, G, R, MODE, 3, 2>, 3);
                default: return go(k_sweep_tma<CW, G, R, MODE, 4, 2>, 4);
                }
            }
        }
        switch (L.stages) {
        case 2: return go(k_sweep_tma<CW, G, R, MODE, 2, 1>, 2);
        case 3: return go(k_sweep_tma<CW, G, R, MODE, 3, 1>, 3);
        default: return go(k_sweep_tma<CW, G, R, MODE, 4, 1>, 4);
        }
    }
    if (L.pair) return cudaErrorInvalidValue;
    k_sweep_owned<CW, G, R, MODE><<<grid, block, 0, st>>>(L);
    return cudaGetLastError();
}

template <int CW, int G, int R>
static int owned_ctas_per_sm_impl(int stages, bool pair)
{
    int n = 0;
    cudaError_t e;
    if (stages >= 2) {
        using Src = SmemSrc<CW, G, R>;
        const int D = stages > 4 ? 4 : stages;
        const int smem = kWarpsPerCta * (D * Src::kStage + 128);
        if (smem > 227 * 1024) return 0;
        auto q = [&](auto kern) {
            cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
            return cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, kern, 32 * kWarpsPerCta, smem);
        };
        if (pair) {
            if (D == 2) e = q(k_sweep_tma<CW, G, R, MODE_J, 2, 2>);
            else if (D == 3) e = q(k_sweep_tma<CW, G, R, MODE_J, 3, 2>);
            else e = q(k_sweep_tma<CW, G, R, MODE_J, 4, 2>);
        } else {
            if (D == 2) e = q(k_sweep_tma<CW, G, R, MODE_J, 2, 1>);
            else if (D == 3) e = q(k_sweep_tma<CW, G, R, MODE_J, 3, 1>);
            else e = q(k_sweep_tma<CW, G, R, MODE_J, 4, 1>);
        }
    } else {
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k_sweep_owned<CW, G, R, MODE_J>, 32 * kWarpsPerCta, 0);
    }
    return e == cudaSuccess ? n : 0;
}

template <int CW, int G>
static int owned_ctas_per_sm_rows(int rows, int stages, bool pair)
{
    switch (rows) {
    case 1: return owned_ctas_per_sm_impl<CW, G, 1>(stages, pair);
    case 2: return owned_ctas_per_sm_impl<CW, G, 2>(stages, pair);
    case 4: return owned_ctas_per_sm_impl<CW, G, 4>(stages, pair);
    }
    return 0;
}

// resident CTAs (of kWarpsPerCta warps) per SM of the J-mode owned kernel; 0 if the configuration cannot launch
int owned_ctas_per_sm(int Nb, int rows, int stages, bool pair)
{
    if (pair && stages < 2) return 0;
    switch (Nb) {
    case 32:  return owned_ctas_per_sm_rows<1, 1>(rows, stages, pair);
    case 64:  return owned_ctas_per_sm_rows<2, 1>(rows, stages, pair);
    case 128: return owned_ctas_per_sm_rows<2, 2>(rows, stages, pair);
    case 256: return owned_ctas_per_sm_rows<2, 4>(rows, stages, pair);
    }
    return 0;
}

template <int CW, int G, int R>
static cudaError_t launch_owned_mode(const SweepLaunch &L, cudaStream_t st)
{
    switch (L.mode) {
    case MODE_J:     return launch_owned_one<CW, G, R, MODE_J>(L, st);
    case MODE_COUNT: return launch_owned_one<CW, G, R, MODE_COUNT>(L, st);
    default:         return launch_owned_one<CW, G, R, MODE_DS>(L, st);
    }
}

template <int CW, int G>
static cudaError_t launch_owned_rows(const SweepLaunch &L, cudaStream_t st)
{
    switch (L.rows) {
    case 1: return launch_owned_mode<CW, G, 1>(L, st);
    case 2: return launch_owned_mode<CW, G, 2>(L, st);
    case 4: return launch_owned_mode<CW, G, 4>(L, st);
    }
    return cudaErrorInvalidValue;
}

cudaError_t launch_sweep_owned(const SweepLaunch &L, cudaStream_t st)
{
    switch (L.Nb) {
    case 32:  return launch_owned_rows<1, 1>(L, st);
    case 64:  return launch_owned_rows<2, 1>(L, st);
    case 128: return launch_owned_rows<2, 2>(L, st);
    case 256: return launch_owned_rows<2, 4>(L, st);
    }
    return cudaErrorInvalidValue;
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
    const float2 *__restrict__ P = L.P + foff;
    float *acc = L.acc + ((long long)slot * L.nbins) * L.ncell + foff;
    const float invL = (MODE == MODE_J) ? D.invL : 1.0f;
    const float Lw = 1.0f / D.invL;
    const bool rev = D.sj < 0;
    float I = L.Ibc[bin];
    const long long U0 = (long long)p * ONE + ONE / 2, V0 = (long long)q * ONE + ONE / 2;
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
                const float2 ks = P[o];
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
template <bool COUNTS>
__global__ void k_finalise(float *__restrict__ J, unsigned *__restrict__ counts, const float2 *__restrict__ Pnat,
                           const float *__restrict__ accN, const float *__restrict__ accNC, int slotsN,
                           const float *__restrict__ accT, const float *__restrict__ accTC, int slotsT,
                           int nx, int ny, int nz, int nbins, float inv_nd, int add_S)
{
    __shared__ float tile[32][33];
    const int bin = blockIdx.z / nz, z = blockIdx.z % nz;
    const int x0 = blockIdx.x * 32, y0 = blockIdx.y * 32;
    const size_t ncell = (size_t)nx * ny * nz;
    const size_t slot_stride = ncell * nbins;
    // transposed layout [x][z][y]: coalesced along y
    for (int dx = threadIdx.y; dx < 32; dx += blockDim.y) {
        const int x = x0 + dx, y = y0 + threadIdx.x;
        float s = 0.0f;
        if (x < nx && y < ny) {
            const size_t i = (size_t)bin * ncell + ((size_t)x * nz + z) * ny + y;
            for (int sl = 0; sl < slotsT; ++sl) s += accT[sl * slot_stride + i] + accTC[sl * slot_stride + i];
        }
        tile[dx][threadIdx.x] = s;
    }
    __syncthreads();
    for (int dy = threadIdx.y; dy < 32; dy += blockDim.y) {
        const int x = x0 + threadIdx.x, y = y0 + dy;
        if (x < nx && y < ny) {
            const size_t i = (size_t)bin * ncell + ((size_t)z * ny + y) * nx + x;
            float s = tile[threadIdx.x][dy];
            for (int sl = 0; sl < slotsN; ++sl) s += accN[sl * slot_stride + i] + accNC[sl * slot_stride + i];
            if (COUNTS) {
                counts[i] = (unsigned)__float2uint_rn(s);
            } else {
                const float2 ks = Pnat[i];
                const float jin = s * inv_nd / ks.x;
                J[i] = add_S ? jin + ks.y : jin;
            }
        }
    }
}

cudaError_t launch_normalise(float *J, const float2 *Pnat, const float *accN, const float *accNC, int slotsN,
                             const float *accT, const float *accTC, int slotsT,
                             int nx, int ny, int nz, int nbins, float inv_nd, int add_S, cudaStream_t st)
{
    dim3 grid((nx + 31) / 32, (ny + 31) / 32, nz * nbins), block(32, 8);
    k_finalise<false><<<grid, block, 0, st>>>(J, nullptr, Pnat, accN, accNC, slotsN, accT, accTC, slotsT,
                                              nx, ny, nz, nbins, inv_nd, add_S);
    return cudaGetLastError();
}

cudaError_t launch_counts_finalise(unsigned *counts, const float *accN, const float *accNC, int slotsN,
                                   const float *accT, const float *accTC, int slotsT,
                                   int nx, int ny, int nz, cudaStream_t st)
{
    dim3 grid((nx + 31) / 32, (ny + 31) / 32, nz), block(32, 8);
    k_finalise<true><<<grid, block, 0, st>>>(nullptr, counts, nullptr, accN, accNC, slotsN, accT, accTC, slotsT,
                                             nx, ny, nz, 1, 1.0f, 0);
    return cudaGetLastError();
}

__device__ __forceinline__ double warp_sum(double v)
{
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// out3 = {sum, min, max} over cells of (acc + accC); out3 must be pre-initialised to {0, +inf, 0}
__global__ void k_ds_reduce(double *out3, const float *__restrict__ acc, const float *__restrict__ accC, long long ncell)
{
    double s = 0.0;
    float mn = 3.0e38f, mx = 0.0f;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < ncell; i += (long long)gridDim.x * blockDim.x) {
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

cudaError_t launch_ds_reduce(double *out3, const float *acc, const float *accC, long long ncell, cudaStream_t st)
{
    int blocks = (int)((ncell + 1023) / 1024);
    if (blocks > 592) blocks = 592;
    k_ds_reduce<<<blocks, 256, 0, st>>>(out3, acc, accC, ncell);
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

}  // namespace rt
