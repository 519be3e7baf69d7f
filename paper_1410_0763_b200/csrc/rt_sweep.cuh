// The owned sweep kernel (k_sweep_tma) of the diffuse-radiation ray sweep, as templates.  Included by
// rt_sweep_nb*.cu, one translation unit per supported width of the memory-contiguous transverse axis
// (so that nvcc compiles them in parallel).
//
// Ownership scheme (replaces the paper's four sequential ray groups):
// one warp owns R consecutive ray rows (transverse axis c) over the full cyclic extent of the
// memory-contiguous transverse axis b: Nb = 32*CW*G columns, each thread owning G chunks of CW
// adjacent columns (aligned vector loads).  Along b the thread owns CELLS: a ray that crosses a
// b-boundary is handed to the owner of the next column (register move / one rotate shuffle per
// chunk; a chunk-to-chunk carry; leaving the last column = leaving the box, and a new ray with the
// inflow intensity enters the first column).  Along c the warp owns RAYS: the memory row of ray
// row r is (q0 + r + shift_k) mod Nc, pure address arithmetic; pieces that fall into the next
// memory row use the next row's data and add to the next row's partial, both held by the same
// thread.  Only the partial of the row above the warp's last ray row (the "seam") has another
// owner; it goes to the seam accumulator accC in global memory with plain stores (or, with the
// handoff, to the next warp of the CTA through a ring in shared memory, announced through an
// mbarrier; rows are processed top-down, so it is ready early in a slab and needed at its end).  Every cell therefore has exactly one writer per accumulator array and launch: no
// atomics on the data path, deterministic sums.
//
// Variants (template parameter V):
//   V = 0  one direction per warp, rays move towards higher memory columns
//   V = 1  one direction per warp, rays move towards lower memory columns (b component reflected):
//          canonical lane / chunk order is the reverse of the memory order
//   V = 2  mirror pair: a direction and its b-mirror share every load, store and exponential
#pragma once
#include "rt_internal.h"

namespace rt {

// ------------------------------------------------------------------------------------------------
// Chunk vectors: the CW adjacent cells a lane owns in one chunk are one value of type VT<CW>::T, and
// every arithmetic step of the segment update acts on the whole chunk.  For CW = 2 these are the
// packed fp32x2 instructions of sm_100a (SASS FFMA2 / FMUL2 / FADD2: two IEEE fp32 results per
// lane and issue slot, each rounded exactly like the scalar instruction).
// ------------------------------------------------------------------------------------------------
template <int CW> struct VT;
template <> struct VT<1> { using T = float;  using D = float2; };    // T: chunk of values / accumulators, D: packed (kappa, S)
template <> struct VT<2> { using T = float2; using D = float4; };

__device__ __forceinline__ float  vmul(float a, float b) { return a * b; }
__device__ __forceinline__ float2 vmul(float2 a, float2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ float  vadd(float a, float b) { return a + b; }
__device__ __forceinline__ float2 vadd(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float  vfma(float a, float b, float c) { return fmaf(a, b, c); }
__device__ __forceinline__ float2 vfma(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
template <class T> __device__ __forceinline__ T vsplat(float s);
template <> __device__ __forceinline__ float  vsplat<float>(float s) { return s; }
template <> __device__ __forceinline__ float2 vsplat<float2>(float s) { return make_float2(s, s); }

__device__ __forceinline__ float ex2_approx(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float  vex2(float t) { return ex2_approx(t); }
__device__ __forceinline__ float2 vex2(float2 t) { return make_float2(ex2_approx(t.x), ex2_approx(t.y)); }
// per element: t > thr ? a : b
__device__ __forceinline__ float  vsel_gt(float t, float thr, float a, float b) { return t > thr ? a : b; }
__device__ __forceinline__ float2 vsel_gt(float2 t, float thr, float2 a, float2 b)
{ return make_float2(t.x > thr ? a.x : b.x, t.y > thr ? a.y : b.y); }

// element of a chunk at memory column 0 / CW-1, and the two ways a b-step moves a chunk's rays:
// towards higher memory columns (a new ray enters column 0) or towards lower ones (enters column CW-1)
__device__ __forceinline__ float vfirst(float v) { return v; }
__device__ __forceinline__ float vfirst(float2 v) { return v.x; }
__device__ __forceinline__ float vlast(float v) { return v; }
__device__ __forceinline__ float vlast(float2 v) { return v.y; }
__device__ __forceinline__ void vshift_up(float &v, float in) { v = in; }
__device__ __forceinline__ void vshift_up(float2 &v, float in) { v.y = v.x; v.x = in; }
__device__ __forceinline__ void vshift_down(float &v, float in) { v = in; }
__device__ __forceinline__ void vshift_down(float2 &v, float in) { v.x = v.y; v.y = in; }

// per element: pad-column bit set ? alt : v   (bit 0 = memory element 0 of the chunk)
__device__ __forceinline__ float  vpad(float v, float alt, unsigned m) { return (m & 1u) ? alt : v; }
__device__ __forceinline__ float2 vpad(float2 v, float alt, unsigned m)
{ return make_float2((m & 1u) ? alt : v.x, (m & 2u) ? alt : v.y); }

__device__ __forceinline__ void unpack(const float2 &v, float &kap, float &src) { kap = v.x; src = v.y; }
__device__ __forceinline__ void unpack(const float4 &v, float2 &kap, float2 &src)
{ kap = make_float2(v.x, v.y); src = make_float2(v.z, v.w); }     // pair-packed layout (rt_internal.h)

// ------------------------------------------------------------------------------------------------
// Segment update (eq. 7, eq. 8), fp32
//   A = 1 - exp(-kappa*len); contribution to the cell += I_in * A  (numerator of eq. 11 times kappa*L,
//   see DESIGN.md "Arithmetic"); I_out = I_in * e + S * A with e = exp(-kappa*len).
// e and A each keep a small RELATIVE error: behind an opaque cell the transmitted part I*e is all that is left, so
// there e comes straight from ex2 (bias-corrected) and A = 1 - e; on thin pieces 1 - e would cancel, so A comes from
// a polynomial and e = 1 - A.
// With t = kappa * ct, ct = -len*log2(e):  e = 2^t,  x = kappa*len = -t*ln2, and for x < 1/4
//   A = x (c0 + c1 x + c2 x^2 + c3 x^3)  (fitted on [0, 1/4], rel. error 3.4e-7)
//     = t (d0 + d1 t + d2 t^2 + d3 t^3),  d_k = c_k (-ln 2)^(k+1).
// ------------------------------------------------------------------------------------------------
template <class T>
__device__ __forceinline__ T one_minus_exp(T kap, T ctv, T &e)
{
    constexpr float thr = -0.36067376022224085f;                   // x < 1/4
    const T t = vmul(kap, ctv);
    const T em = vex2(t);
    T p = vfma(t, vsplat<T>(-0.00871029682457447f), vsplat<T>(-0.055303432047367096f));
    p = vfma(t, p, vsplat<T>(-0.24021217226982117f));
    p = vfma(t, p, vsplat<T>(-0.6931470036506653f));
    const T As = vmul(t, p);
    // MUFU.EX2 is biased low (measured on B200: mean -0.3 ... -0.6 ulp, -2e-8 ... -5e-8 relative); over the ~200
    // pieces of a ray through 60 optical depths that is the -5e-6 the deep-shadow cells of C3 were off by
    const T ec = vfma(em, vsplat<T>(kEx2Bias), em);
    const T Ab = vfma(ec, vsplat<T>(-1.0f), vsplat<T>(1.0f));      // 1 - e, one rounding
    const T A = vsel_gt(t, thr, As, Ab);
    // e consistent with A, without a second select: on thick pieces Ab - A = 0 exactly and e = ec; on thin pieces
    // ec >= 1/2, so Ab = 1 - ec exactly and ec + (Ab - As) = RN(1 - As).  A thin medium is then in exact equilibrium
    // at I = S (e + A = 1 to one rounding) instead of drifting by (e + A - 1) / A per piece.
    e = vadd(ec, vadd(Ab, vmul(A, vsplat<T>(-1.0f))));
    return A;
}

// Store of a finished accumulator chunk: the one writer of these cells in this launch and array.  In MODE_OWNERS
// (rt_debug_writer_counts) the store becomes an atomic increment of every element it would have written, so that
// "one writer per cell, accumulator array and launch" can be read back instead of assumed.
template <int MODE> __device__ __forceinline__ void acc_store(float *p, float v)
{
    if (MODE == MODE_OWNERS) atomicAdd(p, 1.0f); else *p = v;
}
template <int MODE> __device__ __forceinline__ void acc_store(float *p, float2 v)
{
    if (MODE == MODE_OWNERS) { atomicAdd(p, 1.0f); atomicAdd(p + 1, 1.0f); }
    else *reinterpret_cast<float2 *>(p) = v;
}

// ND intensities (1, or 2 for a mirror pair) cross the same cell piece: e, A and S*A are shared.
template <int MODE, int ND, class T>
__device__ __forceinline__ void seg_update(T (&I)[ND], T kap, T src, float len, T ctv, T &part)
{
    if (MODE == MODE_J) {
        T e;
        const T A = one_minus_exp<T>(kap, ctv, e);
        const T SA = vmul(src, A);
        if (ND == 2) part = vfma(vadd(I[0], I[ND - 1]), A, part);
        else         part = vfma(I[0], A, part);
#pragma unroll
        for (int d = 0; d < ND; ++d) I[d] = vfma(I[d], e, SA);   // eq. 7
    } else if (MODE == MODE_COUNT) {
        part = vadd(part, vsplat<T>((float)ND));
    } else if (MODE == MODE_DS) {
        part = vadd(part, vsplat<T>((float)ND * len));
    }
}


// The six slab patterns that occur away from exact boundary touches get straight-line code
// (FLC = compile-time flags); anything else runs the same body with run-time flags (FLC < 0).
constexpr int kPatNone = 0;
constexpr int kPatB    = F_SB1 | F_P1;
constexpr int kPatC    = F_SC1 | F_P1;
constexpr int kPatBC   = F_SB1 | F_P1 | F_SC2 | F_P2;
constexpr int kPatCB   = F_SC1 | F_P1 | F_SB2 | F_P2;
constexpr int kPatD    = F_SB1 | F_SC1 | F_P1;

// ------------------------------------------------------------------------------------------------
// mbarrier helpers used inside the slab body (the rest of the TMA helpers are further down)
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@!p bra WAIT_%=;\n\t}"
        :: "r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned bar)
{ asm volatile("mbarrier.arrive.release.cta.shared::cta.b64 _, [%0];" :: "r"(bar) : "memory"); }

// who owns the rows around this warp's tile (warp-uniform)
struct Seam {
    bool first;          // first warp of the CTA: nobody hands a seam partial in (the CTA below wrote it to accC)
    bool last;           // last active warp of the CTA: the seam partial goes to accC in global memory
    // handoff ring (template HO): two slots of one accumulator row per warp boundary, in the producer's block
    unsigned full_out, empty_out, par_empty;   // producer side (if !last): barriers of the slot in use, parity to wait for
    unsigned char *ring_out;                   // this lane's position in that slot
    unsigned full_in, empty_in, par_full;      // consumer side (if !first): the warp below's barriers
    const unsigned char *ring_in;
};

// ------------------------------------------------------------------------------------------------
// One slab for the R ray rows of a warp, rows top-down (r = R-1 ... 0), stage-major within a row:
// every chunk does piece 0, then the step, then piece 1, ... (a mirror pair needs its
// chunk-to-chunk carries in both chunk orders).
//   sp / sa : this lane's position in the warp's row 0 of the stage's packed-field rows / old
//             accumulator rows (shared memory); row r is at + r * kRowP / kRowA, canonical chunk g
//             at a compile-time offset.  Row R is the seam row = row 0 of the next warp (valid only
//             if some piece steps along c).
//   rowp[r] : this lane's position in the global accumulator row of ray row r (r = R: seam
//             accumulator, used by the CTA's last warp).  New accumulator values go straight to
//             global memory (one writer per cell).
//   I[r][g][d] : intensities of the rays currently in the CW columns of chunk g of ray row r,
//             direction d; elements in MEMORY order.
// ------------------------------------------------------------------------------------------------
//
// Multi-bin packed rows (NB > 1; eqs. 22-23: independent bins sharing one geometry): a row holds
// the NB bins of its cells one after the other, [bin][column], so the G chunks of a lane are GB = G / NB chunks per
// bin; one bulk copy per row feeds all bins, and the slab program, the addresses, the barrier wait and the pattern
// dispatch are shared.  Only the ray handoff along b knows about bins: its chunk-to-chunk carry starts anew, with
// that bin's inflow, at every bin.
template <int CW, int G, int R, int MODE, int FLC, int V, int NB>
__device__ __forceinline__ void slab_rows(const unsigned fl_rt, typename VT<CW>::T (&I)[R][G][(V == 2) ? 2 : 1],
                                          const unsigned char *__restrict__ sp, unsigned char *__restrict__ sa,
                                          const float len0, const float len1, const float len2,
                                          const float (&Ib0)[NB], const float (&Ib1)[NB], const float (&Ic)[NB], const float invL,
                                          const int lane, const int lwrap, const unsigned padmask,
                                          float *const (&rowp)[R + 1], const Seam &seam)
{
    using T = typename VT<CW>::T;
    using DV = typename VT<CW>::D;
    constexpr int ND = (V == 2) ? 2 : 1;
    constexpr bool REV = (V == 1);
    constexpr int GB = G / NB;                  // chunks per bin
    constexpr int kRowP = 32 * CW * G * (int)sizeof(float2), kRowA = 32 * CW * G * (int)sizeof(float);
    constexpr unsigned FULL = 0xffffffffu;
    constexpr float LOG2E = 1.4426950408889634f;
    const unsigned fl = (FLC >= 0) ? (unsigned)FLC : fl_rt;
    const T ct0 = vsplat<T>(-len0 * LOG2E), ct1 = vsplat<T>(-len1 * LOG2E), ct2 = vsplat<T>(-len2 * LOG2E);
    const T invLv = vsplat<T>(invL);
    const bool anySC = (fl & (F_SC1 | F_SC2)) != 0;
    // memory chunk of canonical chunk g, as element offsets within a row
#define RT_MG(g) ((((g) / GB) * GB + (REV ? (GB - 1 - (g) % GB) : (g) % GB)) * 32 * CW)
#define RT_OLD(r, g) (*reinterpret_cast<T *>(sa + (r) * kRowA + RT_MG(g) * (int)sizeof(float)))

    T part_hi[G];                 // partial of memory row r + 1
#pragma unroll
    for (int g = 0; g < G; ++g) part_hi[g] = vsplat<T>(0.0f);

#pragma unroll
    for (int r = R - 1; r >= 0; --r) {
        const bool wrap_r = (r == lwrap);
        T part_lo[G];             // partial of memory row r
        T kc[G], sc[G], kn[G], sn[G];
#pragma unroll
        for (int g = 0; g < G; ++g) {
            unpack(*reinterpret_cast<const DV *>(sp + r * kRowP + RT_MG(g) * (int)sizeof(float2)), kc[g], sc[g]);
            if (anySC)
                unpack(*reinterpret_cast<const DV *>(sp + (r + 1) * kRowP + RT_MG(g) * (int)sizeof(float2)), kn[g], sn[g]);
            else { kn[g] = kc[g]; sn[g] = sc[g]; }
            part_lo[g] = vsplat<T>(0.0f);
        }
        T (&Ir)[G][ND] = I[r];
#pragma unroll
        for (int g = 0; g < G; ++g) seg_update<MODE, ND, T>(Ir[g], kc[g], sc[g], len0, ct0, part_lo[g]);
        bool sel = false;
#pragma unroll
        for (int stage = 1; stage <= 2; ++stage) {
            const unsigned fsb = (stage == 1) ? F_SB1 : F_SB2;
            const unsigned fsc = (stage == 1) ? F_SC1 : F_SC2;
            const unsigned fp = (stage == 1) ? F_P1 : F_P2;
            const float len = (stage == 1) ? len1 : len2;
            const T ct = (stage == 1) ? ct1 : ct2;
            if (fl & (fsb | fsc)) {
                if (MODE == MODE_J) {
                    if (fl & fsb) {
                        // direction 0: hand every ray to the owner of the next column in canonical order
                        // (canonical lane + 1 is always the physical lane + 1); a new ray enters at
                        // canonical column 0.  Within a chunk, memory element 0 is upstream unless REV.
                        float carry = 0.0f;
#pragma unroll
                        for (int g = 0; g < G; ++g) {
                            if (g % GB == 0) carry = Ib0[g / GB];    // inflow of the side face direction 0 enters through
                            const float out = REV ? vfirst(Ir[g][0]) : vlast(Ir[g][0]);
                            const float t = __shfl_sync(FULL, out, (lane + 31) & 31);
                            const float in = (lane == 0) ? carry : t;
                            carry = t;
                            if (REV) vshift_down(Ir[g][0], in);
                            else     vshift_up(Ir[g][0], in);
                        }
                        if (ND == 2) {
                            // mirrored direction: towards lower columns; a new ray enters the last column
#pragma unroll
                            for (int g = G - 1; g >= 0; --g) {
                                if (g % GB == GB - 1) carry = Ib1[g / GB];   // the mirror image enters through the opposite face
                                const float t = __shfl_sync(FULL, vfirst(Ir[g][ND - 1]), (lane + 1) & 31);
                                const float in = (lane == 31) ? carry : t;
                                carry = t;
                                vshift_down(Ir[g][ND - 1], in);
                            }
                        }
                    }
                    if ((fl & fsc) && wrap_r) {   // step along c out of the box: new rays enter
#pragma unroll
                        for (int g = 0; g < G; ++g)
#pragma unroll
                            for (int d = 0; d < ND; ++d)           // pad columns hold rays that have yet to cross the b face
                                Ir[g][d] = vpad(vsplat<T>(Ic[g / GB]), d == 0 ? Ib0[g / GB] : Ib1[g / GB], (padmask >> ((g % GB) * CW)) & 3u);
                    }
                }
                if (fl & fsc) sel = true;
            }
            if (fl & fp) {
#pragma unroll
                for (int g = 0; g < G; ++g) {
                    if (sel) seg_update<MODE, ND, T>(Ir[g], kn[g], sn[g], len, ct, part_hi[g]);
                    else     seg_update<MODE, ND, T>(Ir[g], kc[g], sc[g], len, ct, part_lo[g]);
                }
            }
        }
        // memory row r + 1 is complete: its own pieces (previous iteration) + the pieces of ray row r
        // that stepped along c
        if (r == R - 1) {
            if (anySC) {
                if (seam.last) {
                    // the row above the CTA's tile has another owner: seam accumulator, plain stores
#pragma unroll
                    for (int g = 0; g < G; ++g)
                        acc_store<MODE>(rowp[R] + RT_MG(g), vfma(part_hi[g], invLv, RT_OLD(R, g)));
                } else {
                    // row 0 of the next warp: put the partial into the handoff ring and announce it (the slot is
                    // free once that warp has taken the partial of two stepping slabs ago)
                    mbar_wait(seam.empty_out, seam.par_empty);
#pragma unroll
                    for (int g = 0; g < G; ++g)
                        *reinterpret_cast<T *>(seam.ring_out + RT_MG(g) * (int)sizeof(float)) = vmul(part_hi[g], invLv);
                    __syncwarp();
                    if (lane == 0) mbar_arrive(seam.full_out);
                }
            }
        } else {
#pragma unroll
            for (int g = 0; g < G; ++g)
                acc_store<MODE>(rowp[r + 1] + RT_MG(g), vfma(part_hi[g], invLv, RT_OLD(r + 1, g)));
        }
#pragma unroll
        for (int g = 0; g < G; ++g) part_hi[g] = part_lo[g];
    }
    // memory row 0: own pieces (+ with the handoff the seam partial of the warp below)
    if (anySC && !seam.first) {
        mbar_wait(seam.full_in, seam.par_full);
#pragma unroll
        for (int g = 0; g < G; ++g)
            acc_store<MODE>(rowp[0] + RT_MG(g),
                            vadd(vfma(part_hi[g], invLv, RT_OLD(0, g)), *reinterpret_cast<const T *>(seam.ring_in + RT_MG(g) * (int)sizeof(float))));
        __syncwarp();
        if (lane == 0) mbar_arrive(seam.empty_in);
    } else {
#pragma unroll
        for (int g = 0; g < G; ++g)
            acc_store<MODE>(rowp[0] + RT_MG(g), vfma(part_hi[g], invLv, RT_OLD(0, g)));
    }
#undef RT_OLD
#undef RT_MG
}

#define RT_DISPATCH_SLAB(fl, ...)                                                         \
    switch (fl) {                                                                         \
    case kPatNone: slab_rows<CW, G, R, MODE, kPatNone, V, NB>(__VA_ARGS__); break;        \
    case kPatB:    slab_rows<CW, G, R, MODE, kPatB, V, NB>(__VA_ARGS__); break;           \
    case kPatC:    slab_rows<CW, G, R, MODE, kPatC, V, NB>(__VA_ARGS__); break;           \
    case kPatBC:   slab_rows<CW, G, R, MODE, kPatBC, V, NB>(__VA_ARGS__); break;          \
    case kPatCB:   slab_rows<CW, G, R, MODE, kPatCB, V, NB>(__VA_ARGS__); break;          \
    case kPatD:    slab_rows<CW, G, R, MODE, kPatD, V, NB>(__VA_ARGS__); break;           \
    default:       slab_rows<CW, G, R, MODE, -1, V, NB>(__VA_ARGS__); break;              \
    }

// ------------------------------------------------------------------------------------------------
// TMA / mbarrier helpers (1-D bulk async copies: a mesh row is one contiguous run, so the 1-D bulk
// form of TMA is used rather than tensor maps)
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count)
{ asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(bar), "r"(count) : "memory"); }
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes)
{ asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(bar), "r"(bytes) : "memory"); }
__device__ __forceinline__ void bulk_g2s(unsigned dst, const void *src, unsigned bytes, unsigned bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 :: "r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}

// One lane of a converged warp, chosen by the hardware: inside `if (elect_one())` the compiler knows that a single
// thread is active, so a bulk copy is one ELECT-predicated UBLKCP instead of a loop over the active lanes (which is
// what `if (lane == 0)` around the asm statement compiles to: 15 instructions per copy).
__device__ __forceinline__ bool elect_one()
{
    unsigned pred;
    asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(pred));
    return pred != 0;
}

// flags word of a slab program (rt_internal.h SlabProg): traversal flags | row shift << kShiftBit.  A volatile asm
// load keeps its place at the top of the slab, a whole slab body ahead of its use by the producer.
__device__ __forceinline__ unsigned ld_flags(const SlabProg *p)
{
    unsigned v;
    asm volatile("ld.global.nc.u32 %0, [%1];" : "=r"(v) : "l"(&p->flags));
    return v;
}

// Shared memory of a warp: D stages, each the packed-field rows and the old accumulator rows of one
// slab for the warp's R ray rows plus the seam row above them; then the warp's mbarriers.
template <int CW, int G, int R, int D>
struct StageGeom {
    static constexpr int kNb = 32 * CW * G;
    static constexpr int kRowP = kNb * (int)sizeof(float2);
    static constexpr int kRowA = kNb * (int)sizeof(float);
    static constexpr int kStage = (R + 1) * (kRowP + kRowA);
    static constexpr int kBarFull = D * kStage;               // D mbarriers: stage filled (transaction bytes)
    static constexpr int kBarHand = kBarFull + 32;            // 2 mbarriers: handoff ring slot h holds this warp's seam partial
    static constexpr int kBarEmpty = kBarHand + 32;           // 2 mbarriers: the next warp has taken slot h's partial
    static constexpr int kProg = D * kStage + 128;            // D slab programs (16 B each): slab k's travels with its stage
    static constexpr int kWarpBytes = D * kStage + 128 + 64;
    static_assert(D <= 4, "barrier block holds 4 stages");
};

// Each warp owns a private ring of D stages; stage (k mod D) holds slab k's packed field rows and old
// accumulator rows, copied by bulk async copies (SASS UBLKCP) issued by lane 0 D slabs ahead and
// tracked by one mbarrier per stage (transaction-byte count).  No registers are spent on data in
// flight, so the prefetch depth is set by shared memory.  With HO (rt_tune "handoff") warp w hands
// the seam partial of a slab with a step along c to warp w + 1 through a two-slot ring in shared
// memory (its own unused seam-accumulator rows) instead of the seam accumulator in global memory:
// only the CTA's last warp still reads and writes accC.  The producer may run two stepping slabs
// ahead of its consumer; the consumer never waits unless it has caught up.
template <int CW, int G, int R, int MODE, int D, int V, int W, bool HO, int NB = 1>
__global__ void __launch_bounds__(32 * W)
k_sweep_tma(const SweepLaunch L)
{
    static_assert(G % NB == 0 && (NB == 1 || !HO), "NB bins per row; the seam handoff exists for single-bin rows only");
    constexpr int GB = G / NB;
    using SG = StageGeom<CW, G, R, D>;
    using T = typename VT<CW>::T;
    constexpr int ND = (V == 2) ? 2 : 1;
    constexpr bool REV = (V == 1);
    extern __shared__ __align__(128) unsigned char smem_raw[];

    // warp index through a shuffle from lane 0: provably warp-uniform for the compiler, so that the address arithmetic of
    // the bulk copies (issued by one lane) runs on the uniform datapath instead of being moved there value by value
    const int lane = threadIdx.x & 31, wid = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
    // A launch is a range of work items (entry, row tile) of a list of entries (directions or mirror pairs)
    // that need not end on an entry boundary, so that every launch fills all resident CTA slots.  An entry's
    // accumulators are those of slot = entry mod nslots; nslots exceeds the entries a launch can touch.
    const int item = (int)blockIdx.x + L.item0;
    const int ent = item / L.tiles, tile = item - ent * L.tiles;
    const int slot = ent % L.nslots, bin = blockIdx.z * NB;      // first bin of this CTA's group of NB packed bins
    const DirDev *__restrict__ Dp = L.dirs + L.batch[ent];
    const int Nc = Dp->Nc, Na = Dp->Na;
    const int q0c = tile * (W * R);                              // first ray row of the CTA (L.tiles of them cover Nc)
    const int nact = min(W, (Nc - q0c) / R);                     // warps of this CTA that own rows (Nc % R == 0)
    const int q0 = q0c + wid * R;
    const int sk = (int)Dp->sk * NB, sl = (int)Dp->sl * NB;      // |offsets| < 2^31: checked by rt_create (rows hold NB bins)
    const float invL = (MODE == MODE_J) ? Dp->invL : 1.0f;
    // inflow of the faces this slot's rays enter through (DirDev::layout carries the face indices)
    const int fcs = Dp->layout;
    float Ia[NB], Ib0[NB], Ib1[NB], Ic[NB];
#pragma unroll
    for (int b = 0; b < NB; ++b) {
        const float *__restrict__ Ibin = L.Ibc + 6 * (bin + b);
        Ia[b] = Ibin[(fcs >> 8) & 7]; Ib0[b] = Ibin[(fcs >> 12) & 7]; Ib1[b] = Ibin[((fcs >> 12) & 7) ^ 1]; Ic[b] = Ibin[(fcs >> 16) & 7];
    }
    const SlabProg *__restrict__ prog = L.prog + Dp->prog_off;

    const long long foff = (long long)bin * L.ncell + Dp->base * NB;
    const float2 *__restrict__ P = L.P + foff;
    float *__restrict__ acc = L.acc + ((long long)slot * L.nbins) * L.ncell + foff;
    float *__restrict__ accC = L.accC + ((long long)slot * L.nbins) * L.ncell + foff;

    unsigned char *wbase = smem_raw + wid * SG::kWarpBytes;
    const unsigned wbase_s = smem_u32(wbase);
    const unsigned bars = wbase_s + SG::kBarFull;
    if (lane == 0) {
#pragma unroll
        for (int s = 0; s < D; ++s) mbar_init(bars + 8 * s, 1);
#pragma unroll
        for (int h = 0; h < 2; ++h) { mbar_init(wbase_s + SG::kBarHand + 8 * h, 1); mbar_init(wbase_s + SG::kBarEmpty + 8 * h, 1); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();                                             // every warp's barriers exist before a neighbour touches them
    if (wid >= nact) return;

    Seam seam;
    seam.first = !HO || (wid == 0);
    seam.last = !HO || (wid == nact - 1);

    // producer (lane 0): ask the TMA engine for the rows of the slab described by `ps` into stage s.
    // The seam row's old accumulator is needed only by the CTA's last warp (the others add their seam
    // partial into the next warp's stage).
    // An entry that is the first user of its slot in this sweep starts from zero: its old accumulator rows are not
    // copied (the slot was not cleared either, rt_api.cu); the staging rows are zeroed once instead.
    const bool fresh = (MODE == MODE_J) && ent < L.fresh_below;
    if (fresh) {
#pragma unroll
        for (int s = 0; s < D; ++s)
            for (int i = lane; i < R * SG::kRowA / 16; i += 32)
                *reinterpret_cast<float4 *>(wbase + s * SG::kStage + (R + 1) * SG::kRowP + 16 * i) = make_float4(0.f, 0.f, 0.f, 0.f);
        __syncwarp();
    }
    // Row bookkeeping of one march comes from the slab programs: the flags word of slab k carries, above the traversal
    // flags, the row shift floor(v0 + k m_c) mod Nc (rt_kernels.cu k_build_programs), so the memory row of the first
    // ray row at slab k is (q0 + shift) mod Nc, and the rays step along c inside the slab iff an SC flag is set.
    int poffk = 0;                                               // element offset of the slab being produced (k * sk)
    auto produce = [&](int s, int kp, unsigned fw) {
        if (elect_one()) {
            const unsigned st = wbase_s + s * SG::kStage, bar = bars + 8 * s;
            const bool stp = (fw & (F_SC1 | F_SC2)) != 0;
            int lb = q0 + (int)(fw >> kShiftBit); if (lb >= Nc) lb -= Nc;
            const int nP = (MODE == MODE_J) ? R + (stp ? 1 : 0) : 0;
            const bool seamA = stp && seam.last;
            mbar_expect_tx(bar, (unsigned)(sizeof(SlabProg) + nP * SG::kRowP + ((fresh ? 0 : R) + (seamA ? 1 : 0)) * SG::kRowA));
            bulk_g2s(wbase_s + SG::kProg + (unsigned)sizeof(SlabProg) * s, prog + kp, (unsigned)sizeof(SlabProg), bar);
#pragma unroll
            for (int r = 0; r <= R; ++r) {
                int l = lb + r; if (l >= Nc) l -= Nc;
                const int o = poffk + l * sl;
                // packed rows: 2 floats per cell in either packed layout, rows start at even cells
                if (r < nP) bulk_g2s(st + r * SG::kRowP, P + o, SG::kRowP, bar);
                if (r < R ? !fresh : seamA)
                    bulk_g2s(st + (R + 1) * SG::kRowP + r * SG::kRowA, (r < R ? acc : accC) + o, SG::kRowA, bar);
            }
        }
        poffk += sk;
    };
    unsigned fwq[D];                                             // flags words of the slabs in flight, oldest first
#pragma unroll
    for (int kk = 0; kk < D; ++kk) {
        fwq[kk] = 0;
        if (kk < Na) { fwq[kk] = ld_flags(prog + kk); produce(kk, kk, fwq[kk]); }
    }

    // Rows narrower than the template width are padded (rt_api.cu): a pad column carries a ray that has not yet
    // crossed the b side face (it matters for rays moving towards lower columns, which cross the pad first), so
    // it always holds that face's inflow: at the start and after a row wrap.
    unsigned padmask = 0;
#pragma unroll
    for (int g = 0; g < GB; ++g)                                  // the same for every bin
#pragma unroll
        for (int i = 0; i < CW; ++i)
            if (CW * (REV ? 31 - lane : lane) + i + (REV ? (GB - 1 - g) : g) * 32 * CW >= Dp->Nb) padmask |= 1u << (g * CW + i);
    T I[R][G][ND];
#pragma unroll
    for (int r = 0; r < R; ++r)
#pragma unroll
        for (int g = 0; g < G; ++g)
#pragma unroll
            for (int d = 0; d < ND; ++d) I[r][g][d] = vpad(vsplat<T>(Ia[g / GB]), d == 0 ? Ib0[g / GB] : Ib1[g / GB], (padmask >> ((g % GB) * CW)) & 3u);

    // this lane's first memory column (canonical chunk 0 is memory chunk G-1 when REV)
    const int lcol = CW * (REV ? 31 - lane : lane);
    const unsigned char *lane_p = wbase + lcol * (int)sizeof(float2);
    unsigned char *lane_a = wbase + (R + 1) * SG::kRowP + lcol * (int)sizeof(float);
    float *const acc_l = acc + lcol;
    float *const accC_l = accC + lcol;
    unsigned hcnt = 0;                   // slabs with a step along c so far: handoff ring slot = hcnt & 1, use = hcnt >> 1

    int coffk = 0;                                               // element offset of the current slab
    int s = 0;
    unsigned phase = 0;

#pragma unroll 1
    for (int k = 0; k < Na; ++k) {
        // flags word of the slab this iteration's copies are for: loaded now, used after the slab body
        unsigned fwn = 0;
        if (k + D < Na) fwn = ld_flags(prog + k + D);
        const unsigned fw = fwq[0];
        const unsigned fl = fw & kFlagMask;
        float *rowp[R + 1];
        int lb = q0 + (int)(fw >> kShiftBit); if (lb >= Nc) lb -= Nc;
#pragma unroll
        for (int r = 0; r <= R; ++r) {
            int l = lb + r; if (l >= Nc) l -= Nc;
            rowp[r] = (r < R ? acc_l : accC_l) + (coffk + l * sl);
        }
        const int lwrap = Nc - 1 - lb;
        const unsigned char *sp = lane_p + s * SG::kStage;
        unsigned char *sa = lane_a + s * SG::kStage;
        const bool anySC = (fl & (F_SC1 | F_SC2)) != 0;
        if (HO && anySC) {
            // ring slot of this stepping slab: the (unused) seam accumulator row of stage h in the producer's block
            const unsigned h = hcnt & 1u, use = (hcnt >> 1) & 1u;
            seam.full_out = wbase_s + SG::kBarHand + 8 * h;
            seam.empty_out = wbase_s + SG::kBarEmpty + 8 * h;
            seam.par_empty = use ^ 1u;                           // first use of a slot: passes at once
            seam.ring_out = lane_a + h * SG::kStage + R * SG::kRowA;
            seam.full_in = seam.full_out - SG::kWarpBytes;
            seam.empty_in = seam.empty_out - SG::kWarpBytes;
            seam.par_full = use;
            seam.ring_in = seam.ring_out - SG::kWarpBytes;
            ++hcnt;
        }
        mbar_wait(bars + 8 * s, phase);
        // piece lengths of this slab: they came with the stage (one 16-byte bulk copy), every lane reads the same address
        const float4 prv = *reinterpret_cast<const float4 *>(wbase + SG::kProg + sizeof(SlabProg) * s);
        const float len0 = prv.x, len1 = prv.y, len2 = prv.z;
        RT_DISPATCH_SLAB(fl, fl, I, sp, sa, len0, len1, len2, Ib0, Ib1, Ic, invL, lane, lwrap, padmask, rowp, seam)
        __syncwarp();                     // every lane is done with stage s
        if (k + D < Na) {
            // (measured without this fence: C3 / C4 / C5 unchanged to 0.5 %, so the ordering is kept explicit)
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            produce(s, k + D, fwn);
        }
#pragma unroll
        for (int i = 0; i + 1 < D; ++i) fwq[i] = fwq[i + 1];
        fwq[D - 1] = fwn;
        coffk += sk;
        if (++s == D) { s = 0; phase ^= 1u; }
    }
}

// ------------------------------------------------------------------------------------------------
// Launchers for one width Nb = 32*CW*G (instantiated in rt_sweep_nb*.cu)
// ------------------------------------------------------------------------------------------------
constexpr int kW = kOwnedWarpsPerCta;

template <int CW, int G, int R, int MODE, int D, int V, bool HO, int NB = 1>
static cudaError_t launch_tma_ho(const SweepLaunch &L, dim3 grid, cudaStream_t st)
{
    constexpr int smem = kW * StageGeom<CW, G, R, D>::kWarpBytes;
    if (smem > 227 * 1024) return cudaErrorInvalidValue;
    auto kern = k_sweep_tma<CW, G, R, MODE, D, V, kW, HO, NB>;
    // the shared-memory opt-in is per kernel and device: set once, not on every launch
    static bool opted_in[64] = {};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64 || !opted_in[dev]) {
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
        if (dev >= 0 && dev < 64) opted_in[dev] = true;
    }
    kern<<<grid, dim3(32 * kW), smem, st>>>(L);
    return cudaGetLastError();
}

template <int CW, int G, int R, int MODE, int D, int V>
static cudaError_t launch_tma(const SweepLaunch &L, dim3 grid, cudaStream_t st)
{
    if constexpr (D == 2) {                       // the handoff ablation exists for the default depth only
        if (L.handoff) return launch_tma_ho<CW, G, R, MODE, D, V, true>(L, grid, st);
    } else {
        if (L.handoff) return cudaErrorInvalidValue;
    }
    return launch_tma_ho<CW, G, R, MODE, D, V, false>(L, grid, st);
}

template <int CW, int G, int R, int MODE, int D>
static cudaError_t launch_variant(const SweepLaunch &L, dim3 grid, cudaStream_t st)
{
    if constexpr (MODE == MODE_J || MODE == MODE_OWNERS) {
        if (L.pair) return launch_tma<CW, G, R, MODE, D, 2>(L, grid, st);
    } else {
        if (L.pair) return cudaErrorInvalidValue;
    }
    return L.rev ? launch_tma<CW, G, R, MODE, D, 1>(L, grid, st) : launch_tma<CW, G, R, MODE, D, 0>(L, grid, st);
}

// NB bins packed per row (rt_sweep_nb*x3.cu): J mode and the writer-count mode, ring depth 2, no seam handoff
template <int CW, int G, int R, int NB>
static cudaError_t launch_rows_packed(const SweepLaunch &L, cudaStream_t st)
{
    if (L.tiles != (L.Nc + kW * R - 1) / (kW * R) || L.nitems < 1 || L.nbins % NB != 0 || L.handoff) return cudaErrorInvalidValue;
    const dim3 grid(L.nitems, 1, L.nbins / NB);
    if (L.mode == MODE_J) {
        if (L.pair) return launch_tma_ho<CW, G, R, MODE_J, 2, 2, false, NB>(L, grid, st);
        return L.rev ? launch_tma_ho<CW, G, R, MODE_J, 2, 1, false, NB>(L, grid, st) : launch_tma_ho<CW, G, R, MODE_J, 2, 0, false, NB>(L, grid, st);
    }
    if (L.mode == MODE_OWNERS) {
        if (L.pair) return launch_tma_ho<CW, G, R, MODE_OWNERS, 2, 2, false, NB>(L, grid, st);
        return L.rev ? launch_tma_ho<CW, G, R, MODE_OWNERS, 2, 1, false, NB>(L, grid, st) : launch_tma_ho<CW, G, R, MODE_OWNERS, 2, 0, false, NB>(L, grid, st);
    }
    return cudaErrorInvalidValue;
}

// G = NB * (chunks per bin); rows per warp 1 or 2
template <int CW, int G, int NB>
cudaError_t launch_sweep_packed(const SweepLaunch &L, cudaStream_t st)
{
    switch (L.rows) {
    case 1: return launch_rows_packed<CW, G, 1, NB>(L, st);
    case 2: return launch_rows_packed<CW, G, 2, NB>(L, st);
    }
    return cudaErrorInvalidValue;
}

template <int CW, int G, int NB>
int ctas_per_sm_packed(int rows, bool pair)
{
    int n = 0;
    auto q = [&](auto kern, int smem) {
        if (smem > 227 * 1024) return cudaErrorInvalidValue;
        cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        return cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, kern, 32 * kW, smem);
    };
    cudaError_t e = cudaErrorInvalidValue;
    if (rows == 1) e = pair ? q(k_sweep_tma<CW, G, 1, MODE_J, 2, 2, kW, false, NB>, kW * StageGeom<CW, G, 1, 2>::kWarpBytes)
                            : q(k_sweep_tma<CW, G, 1, MODE_J, 2, 0, kW, false, NB>, kW * StageGeom<CW, G, 1, 2>::kWarpBytes);
    if (rows == 2) e = pair ? q(k_sweep_tma<CW, G, 2, MODE_J, 2, 2, kW, false, NB>, kW * StageGeom<CW, G, 2, 2>::kWarpBytes)
                            : q(k_sweep_tma<CW, G, 2, MODE_J, 2, 0, kW, false, NB>, kW * StageGeom<CW, G, 2, 2>::kWarpBytes);
    return e == cudaSuccess ? n : 0;
}

template <int CW, int G, int R>
static cudaError_t launch_rows(const SweepLaunch &L, cudaStream_t st)
{
    if (L.tiles != (L.Nc + kW * R - 1) / (kW * R) || L.nitems < 1) return cudaErrorInvalidValue;
    const dim3 grid(L.nitems, 1, L.nbins);
    if (L.mode == MODE_COUNT) return launch_variant<CW, G, R, MODE_COUNT, 2>(L, grid, st);   // diagnostics: depth 2
    if (L.mode == MODE_DS)    return launch_variant<CW, G, R, MODE_DS, 2>(L, grid, st);
    if (L.mode == MODE_OWNERS) return launch_variant<CW, G, R, MODE_OWNERS, 2>(L, grid, st);
    switch (L.stages) {
    case 4:  if constexpr (CW * G <= 2) return launch_variant<CW, G, R, MODE_J, 4>(L, grid, st); else return cudaErrorInvalidValue;   // rows of <= 64 cells
    case 3:  return launch_variant<CW, G, R, MODE_J, 3>(L, grid, st);
    default: return launch_variant<CW, G, R, MODE_J, 2>(L, grid, st);
    }
}

// MAXR: largest number of ray rows per warp instantiated for this width (registers: R * G * CW intensities per direction)
template <int CW, int G, int MAXR = 4>
cudaError_t launch_sweep_nb(const SweepLaunch &L, cudaStream_t st)
{
    switch (L.rows) {
    case 1: return launch_rows<CW, G, 1>(L, st);
    case 2: if constexpr (MAXR >= 2) return launch_rows<CW, G, 2>(L, st); else return cudaErrorInvalidValue;
    case 4: if constexpr (CW * G <= 4) return launch_rows<CW, G, 4>(L, st); else return cudaErrorInvalidValue;   // rows of <= 128 cells
    }
    return cudaErrorInvalidValue;
}

template <int CW, int G, int R, int D>
static int ctas_per_sm_one(bool pair)
{
    constexpr int smem = kW * StageGeom<CW, G, R, D>::kWarpBytes;
    if (smem > 227 * 1024) return 0;
    int n = 0;
    auto q = [&](auto kern) {
        cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        return cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, kern, 32 * kW, smem);
    };
    const cudaError_t e = pair ? q(k_sweep_tma<CW, G, R, MODE_J, D, 2, kW, false>) : q(k_sweep_tma<CW, G, R, MODE_J, D, 0, kW, false>);
    return e == cudaSuccess ? n : 0;
}

template <int CW, int G, int R>
static int ctas_per_sm_rows(int stages, bool pair)
{
    switch (stages) {
    case 4:  if constexpr (CW * G <= 2) return ctas_per_sm_one<CW, G, R, 4>(pair); else return 0;
    case 3:  return ctas_per_sm_one<CW, G, R, 3>(pair);
    default: return ctas_per_sm_one<CW, G, R, 2>(pair);
    }
}

// resident CTAs (of kOwnedWarpsPerCta warps) per SM of the J-mode kernel; 0 if the configuration cannot launch
template <int CW, int G, int MAXR = 4>
int ctas_per_sm_nb(int rows, int stages, bool pair)
{
    switch (rows) {
    case 1: return ctas_per_sm_rows<CW, G, 1>(stages, pair);
    case 2: if constexpr (MAXR >= 2) return ctas_per_sm_rows<CW, G, 2>(stages, pair); else return 0;
    case 4: if constexpr (CW * G <= 4) return ctas_per_sm_rows<CW, G, 4>(stages, pair); else return 0;
    }
    return 0;
}

}  // namespace rt
