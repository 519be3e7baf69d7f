/*
 * oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, double-precision CPU statement of the diffuse-radiation ray sweep of
 * Tanaka, Yoshikawa, Okamoto & Hasegawa (arXiv:1410.0763), written from the paper
 * and the readings listed in DESIGN.md ("Readings").
 * It shares no code with the CUDA library; only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may call it.
 *
 * What it follows, in the paper's order:
 *   PAPER.md:86      "equally spaced parallel rays"                     -> ray lattice  (orc_sweep, O3)
 *   PAPER.md:88-92   eq. (7)  I_out = I_in e^-dtau + S (1 - e^-dtau)    -> segment update (O5)
 *   PAPER.md:94-97   eq. (8)  path-averaged incoming intensity          -> num += ds * I_in * f(dtau)
 *   PAPER.md:105-111 eqs. (10)-(11) multi-ray per-cell average          -> num/den per direction (O6)
 *   PAPER.md:113-119 eqs. (12)-(13) angular mean, J = J_in + S          -> Jin += w * num/den ; J = Jin + S
 *   PAPER.md:183     HEALPix directions, N_d = 12 Nside^2               -> orc_healpix_dirs (O2)
 *   PAPER.md:226     4 ray groups in 3-D never share a cell             -> orc_group_conflicts (pin P9)
 *
 * One ray at a time, no grouping, no blocking, no reordering.  Geometry is exact integer
 * arithmetic (slopes quantised to 2^-20, readings A3/A4); intensities are fp64.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): P1 direction set, P2 axis-aligned hand
 * enumeration, P3 per-cell sum of ds, P5 uniform-slab closed form, P6 optically thin limit,
 * P7 mirror/permutation symmetry, P8 independent fine-step brute force, P9 group ownership,
 * P10 worked example (tests/golden/worked_example.txt), P11 optically thick limit.
 * Beyond those pins the J of the five benchmark configs is "parity unpinned": no external
 * number exists for them; this oracle is the reference.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_F 20
#define ORC_ONE ((int64_t)1 << ORC_F)

typedef struct {
    int a, b, c;        /* dominant axis and the two transverse axes (0=x,1=y,2=z)          */
    int refl[3];        /* refl[axis] = 1 if that axis is mirrored (component < 0)          */
    int64_t Mb, Mc;     /* quantised slopes |n_b|/|n_a|, |n_c|/|n_a| in units of 2^-20      */
    double L;           /* path length per slab in units of cell_width                      */
} orc_dir_t;

/* ---- O2: HEALPix ring-scheme pixel centres (Gorski et al. 2005 closed form) ---- */
int orc_healpix_dirs(int nside, double *dirs /* [12 nside^2][3] */)
{
    if (nside < 1 || !dirs) return -1;
    const double pi = 3.14159265358979323846;
    long n = 0;
    for (int i = 1; i <= 4 * nside - 1; ++i) {
        int npix_ring, ii;
        double z, sgn = 1.0;
        if (i < nside) {                       /* north polar cap */
            ii = i; npix_ring = 4 * ii;
            z = 1.0 - (double)ii * ii / (3.0 * nside * nside);
        } else if (i <= 3 * nside) {           /* equatorial belt */
            ii = i; npix_ring = 4 * nside;
            z = 4.0 / 3.0 - 2.0 * i / (3.0 * nside);
        } else {                               /* south polar cap: mirror of ring 4 nside - i */
            ii = 4 * nside - i; npix_ring = 4 * ii; sgn = -1.0;
            z = 1.0 - (double)ii * ii / (3.0 * nside * nside);
        }
        for (int j = 1; j <= npix_ring; ++j) {
            double phi;
            if (i < nside || i > 3 * nside) {
                phi = (j - 0.5) * pi / (2.0 * ii);
            } else {
                int s = (i - nside + 1) % 2;
                phi = (j - 0.5 * s) * pi / (2.0 * nside);
            }
            double st = sqrt((1.0 - z) * (1.0 + z));
            dirs[3 * n + 0] = st * cos(phi);
            dirs[3 * n + 1] = st * sin(phi);
            dirs[3 * n + 2] = sgn * z;
            ++n;
        }
    }
    return (int)n;
}

/* ---- O2: per-direction record ---- */
int orc_dir_record(const double n[3], int *a_out, int refl_out[3], int64_t *Mb, int64_t *Mc, double *L)
{
    double ax = fabs(n[0]), ay = fabs(n[1]), az = fabs(n[2]);
    if (!(ax > 0.0 || ay > 0.0 || az > 0.0)) return -1;
    int a = 0;                                  /* argmax |n_i|, ties -> lowest axis index (A5) */
    double am = ax;
    if (ay > am) { a = 1; am = ay; }
    if (az > am) { a = 2; am = az; }
    int b = (a == 0) ? 1 : 0;
    int c = (a == 2) ? 1 : 2;
    double mb = fabs(n[b]) / am, mc = fabs(n[c]) / am;    /* in [0,1] */
    int64_t qb = (int64_t)nearbyint(mb * (double)ORC_ONE);
    int64_t qc = (int64_t)nearbyint(mc * (double)ORC_ONE);
    if (qb > ORC_ONE) qb = ORC_ONE;
    if (qc > ORC_ONE) qc = ORC_ONE;
    *a_out = a;
    for (int i = 0; i < 3; ++i) refl_out[i] = (n[i] < 0.0) ? 1 : 0;
    *Mb = qb; *Mc = qc;
    double fb = (double)qb / (double)ORC_ONE, fc = (double)qc / (double)ORC_ONE;
    *L = sqrt(1.0 + fb * fb + fc * fc);
    return 0;
}

static void make_dir(const double n[3], orc_dir_t *d)
{
    orc_dir_record(n, &d->a, d->refl, &d->Mb, &d->Mc, &d->L);
    d->b = (d->a == 0) ? 1 : 0;
    d->c = (d->a == 2) ? 1 : 2;
}

/* f(x) = (1 - e^-x)/x  (eq. 8), O5 */
static double f_of(double x)
{
    if (x < 1e-8) return 1.0 - 0.5 * x;
    return -expm1(-x) / x;
}

typedef struct {
    int dims[3];
    int nbins;
    size_t ncell;
    const float *kappa, *S;     /* [nbins][nz][ny][nx] */
    const double *Ibc;          /* [nbins] or NULL (=0) */
    const double *Ibc6;         /* [nbins][6] per entry face (-x,+x,-y,+y,-z,+z) or NULL: overrides Ibc (A10) */
    double cell_width;
    int rays;                   /* r: rays per cell width in each transverse axis (O3, A13); 0 means 1 */
    /* per-direction scratch (owned by the calling thread) */
    double *num;                /* [nbins][ncell] */
    double *den;                /* [ncell] */
    uint32_t *cnt;              /* [ncell] */
    const int32_t *slot;        /* NULL: accumulate everywhere; else accumulate only where slot[cell] >= 0 */
    int kstop;                  /* > 0: march slabs 0 .. kstop-1 only (orc_sweep_cells: nothing is sampled further downstream) */
    /* optional per-ray outputs for a single direction */
    double *exitI;              /* [nq][np][nbins] */
    double *chord;              /* [nq][np] */
    int pmin, qmin, np, nq;
    /* optional group-conflict check (P9): owner[g][cell] = ray id + 1 */
    int64_t *owner;             /* [4][ncell] or NULL */
    long conflicts;
    /* segment tally */
    unsigned long long nseg;
} orc_work_t;

/* one segment of one ray: O5 */
static inline void do_segment(orc_work_t *w, size_t cell, double ds, double *I)
{
    if (!w->slot || w->slot[cell] >= 0) {
        w->den[cell] += ds;
        w->cnt[cell] += 1;
    }
    w->nseg += 1;
    for (int bin = 0; bin < w->nbins; ++bin) {
        size_t o = (size_t)bin * w->ncell + cell;
        double dtau = (double)w->kappa[o] * ds;
        if (!w->slot || w->slot[cell] >= 0)
            w->num[o] += ds * I[bin] * f_of(dtau);                       /* eq. 8 weighted by ds (A7) */
        I[bin] = I[bin] * exp(-dtau) + (double)w->S[o] * (-expm1(-dtau));  /* eq. 7, term by term */
    }
}

/* O3-O4: march one lattice ray (p,q) of direction d through all slabs */
static void trace_ray(orc_work_t *w, const orc_dir_t *d, int64_t p, int64_t q)
{
    const int Na = w->dims[d->a], Nb = w->dims[d->b], Nc = w->dims[d->c];
    const int64_t ONE = ORC_ONE;
    /* O3: lattice of spacing 1/r; ray (p,q) meets the plane a = 0 at U0 = (2p+1) ONE/(2r), V0 = (2q+1) ONE/(2r)
       (r divides 2^19, checked by the callers; r = 1: cell-centre offsets, A2) */
    const int64_t r_ = w->rays > 0 ? w->rays : 1;
    const int64_t U0 = (2 * p + 1) * (ONE / (2 * r_)), V0 = (2 * q + 1) * (ONE / (2 * r_));
    const double Lw = d->L * w->cell_width;
    double I[16];
    for (int bin = 0; bin < w->nbins; ++bin) I[bin] = w->Ibc ? w->Ibc[bin] : 0.0;
    if (w->Ibc6) {
        /* A10: the ray starts with the inflow of the face through which it enters the box, i.e. the
           face it crosses last: the a-face if it starts inside the transverse extent, else the side
           face (b or c) whose plane it reaches later (exact integers; both at once: c). */
        const int64_t j0 = U0 >> ORC_F, l0 = V0 >> ORC_F;
        int ax;
        if (j0 >= 0 && l0 >= 0) ax = d->a;
        else if (j0 >= 0) ax = d->c;
        else if (l0 >= 0) ax = d->b;
        else ax = ((-V0) * d->Mb >= (-U0) * d->Mc) ? d->c : d->b;
        const int face = 2 * ax + (d->refl[ax] ? 1 : 0);            /* marching towards -axis enters through the + face */
        for (int bin = 0; bin < w->nbins; ++bin) I[bin] = w->Ibc6[6 * bin + face];
    }
    double chord = 0.0;
    size_t stride[3] = {1, (size_t)w->dims[0], (size_t)w->dims[0] * w->dims[1]};

    const int kend = (w->kstop > 0 && w->kstop < Na) ? w->kstop : Na;
    for (int k = 0; k < kend; ++k) {
        int64_t U = U0 + (int64_t)k * d->Mb, V = V0 + (int64_t)k * d->Mc;
        int64_t j = U >> ORC_F, l = V >> ORC_F;                      /* floor */
        if (j < -1 || j >= Nb || l < -1 || l >= Nc) continue;        /* whole slab outside the box */
        int64_t Db = (j + 1) * ONE - U, Dc = (l + 1) * ONE - V;      /* distance to next boundary, >= 1 */
        int crossb = (U + d->Mb > (j + 1) * ONE);                    /* strict (A3) */
        int crossc = (V + d->Mc > (l + 1) * ONE);
        /* pieces: up to 3, [t_s, t_{s+1}] with cell offsets */
        double t[4]; int dj[3], dl[3]; int np = 0;
        t[0] = 0.0;
        if (!crossb && !crossc) {
            dj[0] = 0; dl[0] = 0; t[1] = 1.0; np = 1;
        } else if (crossb && !crossc) {
            dj[0] = 0; dl[0] = 0; t[1] = (double)Db / (double)d->Mb;
            dj[1] = 1; dl[1] = 0; t[2] = 1.0; np = 2;
        } else if (!crossb && crossc) {
            dj[0] = 0; dl[0] = 0; t[1] = (double)Dc / (double)d->Mc;
            dj[1] = 0; dl[1] = 1; t[2] = 1.0; np = 2;
        } else {
            int64_t lhs = Db * d->Mc, rhs = Dc * d->Mb;              /* t_b ? t_c  <=>  Db*Mc ? Dc*Mb */
            double tb = (double)Db / (double)d->Mb, tc = (double)Dc / (double)d->Mc;
            if (lhs < rhs) {            /* b first */
                dj[0] = 0; dl[0] = 0; t[1] = tb;
                dj[1] = 1; dl[1] = 0; t[2] = tc;
                dj[2] = 1; dl[2] = 1; t[3] = 1.0; np = 3;
            } else if (lhs > rhs) {     /* c first */
                dj[0] = 0; dl[0] = 0; t[1] = tc;
                dj[1] = 0; dl[1] = 1; t[2] = tb;
                dj[2] = 1; dl[2] = 1; t[3] = 1.0; np = 3;
            } else {                    /* simultaneous: one diagonal step */
                dj[0] = 0; dl[0] = 0; t[1] = tb;
                dj[1] = 1; dl[1] = 1; t[2] = 1.0; np = 2;
            }
        }
        for (int s = 0; s < np; ++s) {
            int64_t jj = j + dj[s], ll = l + dl[s];
            if (jj < 0 || jj >= Nb || ll < 0 || ll >= Nc) continue;  /* outside the box */
            if (!(t[s + 1] > t[s])) continue;                        /* zero-length piece dropped */
            double ds = (t[s + 1] - t[s]) * Lw;
            int idx[3];
            idx[d->a] = d->refl[d->a] ? Na - 1 - k : k;
            idx[d->b] = d->refl[d->b] ? Nb - 1 - (int)jj : (int)jj;
            idx[d->c] = d->refl[d->c] ? Nc - 1 - (int)ll : (int)ll;
            size_t cell = idx[0] * stride[0] + idx[1] * stride[1] + idx[2] * stride[2];
            if (w->owner) {
                int g = (int)(((p % 2) + 2) % 2) + 2 * (int)(((q % 2) + 2) % 2);
                int64_t id = (q - w->qmin) * (int64_t)w->np + (p - w->pmin) + 1;
                int64_t *o = &w->owner[(size_t)g * w->ncell + cell];
                if (*o != 0 && *o != id) w->conflicts += 1;
                *o = id;
            }
            do_segment(w, cell, ds, I);
            chord += ds;
        }
    }
    if (w->exitI) {
        size_t r = (size_t)(q - w->qmin) * w->np + (size_t)(p - w->pmin);
        for (int bin = 0; bin < w->nbins; ++bin) w->exitI[r * w->nbins + bin] = I[bin];
        if (w->chord) w->chord[r] = chord;
    }
}

static void lattice_range(const int dims[3], const orc_dir_t *d, int *pmin, int *qmin)
{
    const int Na = dims[d->a];
    /* O3: p from -ceil(Na*Mb/ONE)-1 to Nb-1 */
    *pmin = -(int)((Na * d->Mb + ORC_ONE - 1) / ORC_ONE) - 1;
    *qmin = -(int)((Na * d->Mc + ORC_ONE - 1) / ORC_ONE) - 1;
}

/* all rays of one direction, lattice order (q outer, p inner) */
static void sweep_direction(orc_work_t *w, const orc_dir_t *d)
{
    int pmin, qmin;
    lattice_range(w->dims, d, &pmin, &qmin);
    w->pmin = pmin; w->qmin = qmin;
    w->np = w->dims[d->b] - pmin; w->nq = w->dims[d->c] - qmin;
    const int64_t r_ = w->rays > 0 ? w->rays : 1;                  /* O3: p from r*pmin to r*Nb - 1, q likewise */
    for (int64_t q = r_ * qmin; q < r_ * w->dims[d->c]; ++q)
        for (int64_t p = r_ * pmin; p < r_ * w->dims[d->b]; ++p)
            trace_ray(w, d, p, q);
}

/*
 * Full sweep (O1-O7).  All pointers are host pointers.  Optional outputs may be NULL.
 *   kappa, S   : fp32 [nbins][nz][ny][nx], widened to fp64 inside
 *   dirs       : fp64 [ndirs][3]
 *   Ibc        : fp64 [nbins] boundary inflow, NULL = 0
 *   Jin, J     : fp64 [nbins][nz][ny][nx]   (eq. 13 and eq. 12)
 *   sum_ds     : fp64 [ndirs]               sum of ds over all segments of the direction
 *   seg_total  : total number of positive-length in-box segments over all directions
 *   cnt_sum    : uint32 [ncell] per-cell segment count summed over directions
 *   cnt_dirs   : list of ncnt direction indices whose per-cell counts are wanted
 *   cnt_out    : uint32 [ncnt][ncell]
 *   min_den/max_den : fp64 [ndirs] min / max over cells of the per-cell sum of ds (pin P3)
 *   nthreads   : OpenMP threads over directions (<=0: default)
 * Returns 0, or <0 on bad arguments / allocation failure.
 */
int orc_sweep_faces(int nx, int ny, int nz, int nbins, const float *kappa, const float *S, const double *dirs, int ndirs,
                    const double *Ibc, const double *Ibc6, double cell_width, int rays, double *Jin, double *J,
                    double *sum_ds, unsigned long long *seg_total, uint32_t *cnt_sum, const int *cnt_dirs, int ncnt,
                    uint32_t *cnt_out, double *min_den, double *max_den, int nthreads);

int orc_sweep_rays(int nx, int ny, int nz, int nbins,
              const float *kappa, const float *S,
              const double *dirs, int ndirs, const double *Ibc, double cell_width, int rays,
              double *Jin, double *J, double *sum_ds, unsigned long long *seg_total,
              uint32_t *cnt_sum, const int *cnt_dirs, int ncnt, uint32_t *cnt_out,
              double *min_den, double *max_den, int nthreads)
{
    return orc_sweep_faces(nx, ny, nz, nbins, kappa, S, dirs, ndirs, Ibc, NULL, cell_width, rays, Jin, J, sum_ds,
                           seg_total, cnt_sum, cnt_dirs, ncnt, cnt_out, min_den, max_den, nthreads);
}

/* as orc_sweep_rays, with an inflow intensity per bin and entry face: Ibc6 [nbins][6] or NULL */
int orc_sweep_faces(int nx, int ny, int nz, int nbins,
              const float *kappa, const float *S,
              const double *dirs, int ndirs, const double *Ibc, const double *Ibc6, double cell_width, int rays,
              double *Jin, double *J, double *sum_ds, unsigned long long *seg_total,
              uint32_t *cnt_sum, const int *cnt_dirs, int ncnt, uint32_t *cnt_out,
              double *min_den, double *max_den, int nthreads)
{
    if (nx < 1 || ny < 1 || nz < 1 || nbins < 1 || nbins > 16 || !kappa || !S || !dirs || ndirs < 1) return -1;
    if (rays < 1 || rays > (1 << 19) || (rays & (rays - 1)) != 0) return -1;      /* r must divide 2^(F-1) (O3) */
    const size_t ncell = (size_t)nx * ny * nz;
    int fail = 0;
    unsigned long long total = 0;
    if (Jin) memset(Jin, 0, sizeof(double) * ncell * nbins);
    if (cnt_sum) memset(cnt_sum, 0, sizeof(uint32_t) * ncell);
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
#pragma omp parallel reduction(+ : total)
    {
        orc_work_t w;
        memset(&w, 0, sizeof(w));
        w.dims[0] = nx; w.dims[1] = ny; w.dims[2] = nz;
        w.nbins = nbins; w.ncell = ncell; w.kappa = kappa; w.S = S; w.Ibc = Ibc; w.cell_width = cell_width;
        w.rays = rays; w.Ibc6 = Ibc6;
        w.num = (double *)calloc(ncell * nbins, sizeof(double));
        w.den = (double *)calloc(ncell, sizeof(double));
        w.cnt = (uint32_t *)calloc(ncell, sizeof(uint32_t));
        double *Jloc = Jin ? (double *)calloc(ncell * nbins, sizeof(double)) : NULL;
        uint32_t *cloc = cnt_sum ? (uint32_t *)calloc(ncell, sizeof(uint32_t)) : NULL;
        if (!w.num || !w.den || !w.cnt || (Jin && !Jloc) || (cnt_sum && !cloc)) {
#pragma omp atomic write
            fail = 1;
        } else {
#pragma omp for schedule(dynamic, 1)
            for (int i = 0; i < ndirs; ++i) {
                orc_dir_t d;
                make_dir(&dirs[3 * i], &d);
                w.nseg = 0;
                sweep_direction(&w, &d);
                total += w.nseg;
                /* O6 */
                double sds = 0.0, dmin = INFINITY, dmax = 0.0;
                const double wgt = 1.0 / (double)ndirs;            /* eq. 12-13: plain 1/N_d mean (A11) */
                for (size_t cidx = 0; cidx < ncell; ++cidx) {
                    double dn = w.den[cidx];
                    sds += dn;
                    if (dn < dmin) dmin = dn;
                    if (dn > dmax) dmax = dn;
                    if (dn > 0.0 && Jloc)
                        for (int bin = 0; bin < nbins; ++bin)
                            Jloc[(size_t)bin * ncell + cidx] += wgt * w.num[(size_t)bin * ncell + cidx] / dn;
                    if (cloc) cloc[cidx] += w.cnt[cidx];
                }
                if (sum_ds) sum_ds[i] = sds;
                if (min_den) min_den[i] = dmin;
                if (max_den) max_den[i] = dmax;
                for (int s = 0; s < ncnt; ++s)
                    if (cnt_dirs[s] == i) memcpy(cnt_out + (size_t)s * ncell, w.cnt, sizeof(uint32_t) * ncell);
                memset(w.num, 0, sizeof(double) * ncell * nbins);
                memset(w.den, 0, sizeof(double) * ncell);
                memset(w.cnt, 0, sizeof(uint32_t) * ncell);
            }
#pragma omp critical
            {
                if (Jin) for (size_t o = 0; o < ncell * nbins; ++o) Jin[o] += Jloc[o];
                if (cnt_sum) for (size_t o = 0; o < ncell; ++o) cnt_sum[o] += cloc[o];
            }
        }
        free(w.num); free(w.den); free(w.cnt); free(Jloc); free(cloc);
    }
    if (fail) return -2;
    if (seg_total) *seg_total = total;
    if (J && Jin)                                                   /* eq. 12 */
        for (size_t o = 0; o < ncell * nbins; ++o) J[o] = Jin[o] + (double)S[o];
    return 0;
}

/* r = 1: one ray per cell cross-section (all five configs) */
int orc_sweep(int nx, int ny, int nz, int nbins,
              const float *kappa, const float *S,
              const double *dirs, int ndirs, const double *Ibc, double cell_width,
              double *Jin, double *J, double *sum_ds, unsigned long long *seg_total,
              uint32_t *cnt_sum, const int *cnt_dirs, int ncnt, uint32_t *cnt_out,
              double *min_den, double *max_den, int nthreads)
{
    return orc_sweep_rays(nx, ny, nz, nbins, kappa, S, dirs, ndirs, Ibc, cell_width, 1, Jin, J, sum_ds, seg_total,
                          cnt_sum, cnt_dirs, ncnt, cnt_out, min_den, max_den, nthreads);
}

/*
 * One direction, with per-ray outputs (pin P5) and the 4-group ownership check (pin P9).
 *   exitI : fp64 [nq][np][nbins]; chord : fp64 [nq][np]; lattice = [pmin, Nb) x [qmin, Nc)
 *   lat   : int[4] = {pmin, qmin, np, nq} (always written; call with exitI = NULL to size the buffers)
 *   conflicts : number of (group, cell) pairs visited by two different rays of one group
 */
int orc_trace_direction(int nx, int ny, int nz, int nbins,
                        const float *kappa, const float *S, const double n[3], const double *Ibc,
                        double cell_width, int lat[4], double *exitI, double *chord, long *conflicts)
{
    if (nx < 1 || ny < 1 || nz < 1 || nbins < 1 || nbins > 16 || !kappa || !S || !n || !lat) return -1;
    orc_work_t w;
    memset(&w, 0, sizeof(w));
    w.dims[0] = nx; w.dims[1] = ny; w.dims[2] = nz;
    w.nbins = nbins; w.ncell = (size_t)nx * ny * nz; w.kappa = kappa; w.S = S; w.Ibc = Ibc; w.cell_width = cell_width;
    orc_dir_t d;
    make_dir(n, &d);
    int pmin, qmin;
    lattice_range(w.dims, &d, &pmin, &qmin);
    lat[0] = pmin; lat[1] = qmin; lat[2] = w.dims[d.b] - pmin; lat[3] = w.dims[d.c] - qmin;
    if (!exitI && !conflicts) return 0;
    w.num = (double *)calloc(w.ncell * nbins, sizeof(double));
    w.den = (double *)calloc(w.ncell, sizeof(double));
    w.cnt = (uint32_t *)calloc(w.ncell, sizeof(uint32_t));
    if (conflicts) w.owner = (int64_t *)calloc(4 * w.ncell, sizeof(int64_t));
    if (!w.num || !w.den || !w.cnt || (conflicts && !w.owner)) { free(w.num); free(w.den); free(w.cnt); free(w.owner); return -2; }
    w.exitI = exitI; w.chord = chord;
    sweep_direction(&w, &d);
    if (conflicts) *conflicts = w.conflicts;
    free(w.num); free(w.den); free(w.cnt); free(w.owner);
    return 0;
}

/*
 * J_in at a list of sampled cells, computed one cell set at a time by tracing only the lattice
 * rays that can touch a sampled cell (the same trace_ray as the full sweep).  Used for parity
 * at full benchmark sizes, where the full sweep would take too long on the host.
 *   cells : int [ncells][3] = (x,y,z);  Jin_out / J_out : fp64 [nbins][ncells]
 *   den_out : fp64 [ndirs][ncells] per-cell sum of ds (may be NULL); cnt_out : uint32 [ncells] summed over directions
 */
int orc_sweep_cells(int nx, int ny, int nz, int nbins,
                    const float *kappa, const float *S,
                    const double *dirs, int ndirs, const double *Ibc, double cell_width,
                    const int *cells, int ncells, double *Jin_out, double *J_out,
                    uint32_t *cnt_out, int nthreads)
{
    if (nx < 1 || ny < 1 || nz < 1 || nbins < 1 || nbins > 16 || !kappa || !S || !dirs || ndirs < 1 || !cells || ncells < 1) return -1;
    const size_t ncell = (size_t)nx * ny * nz;
    int32_t *slot = (int32_t *)malloc(sizeof(int32_t) * ncell);
    if (!slot) return -2;
    for (size_t i = 0; i < ncell; ++i) slot[i] = -1;
    for (int s = 0; s < ncells; ++s) {
        const int *c = &cells[3 * s];
        if (c[0] < 0 || c[0] >= nx || c[1] < 0 || c[1] >= ny || c[2] < 0 || c[2] >= nz) { free(slot); return -1; }
        slot[(size_t)c[2] * ny * nx + (size_t)c[1] * nx + c[0]] = s;
    }
    for (size_t o = 0; o < (size_t)ncells * nbins; ++o) Jin_out[o] = 0.0;
    if (cnt_out) memset(cnt_out, 0, sizeof(uint32_t) * ncells);
    int fail = 0;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
#pragma omp parallel
    {
        orc_work_t w;
        memset(&w, 0, sizeof(w));
        w.dims[0] = nx; w.dims[1] = ny; w.dims[2] = nz;
        w.nbins = nbins; w.ncell = ncell; w.kappa = kappa; w.S = S; w.Ibc = Ibc; w.cell_width = cell_width;
        w.slot = slot;
        w.num = (double *)calloc(ncell * nbins, sizeof(double));
        w.den = (double *)calloc(ncell, sizeof(double));
        w.cnt = (uint32_t *)calloc(ncell, sizeof(uint32_t));
        double *Jloc = (double *)calloc((size_t)ncells * nbins, sizeof(double));
        uint32_t *cloc = (uint32_t *)calloc(ncells, sizeof(uint32_t));
        /* the launch lattice of any direction has at most N + N_a + 2 rays along each transverse axis (O3) */
        const size_t nmax = (size_t)(nx > ny ? (nx > nz ? nx : nz) : (ny > nz ? ny : nz));
        int32_t *seen = (int32_t *)calloc((2 * nmax + 2) * (2 * nmax + 2), sizeof(int32_t));
        int32_t *stamp = (int32_t *)calloc((2 * nmax + 2) * (2 * nmax + 2), sizeof(int32_t));
        int32_t *cand_p = (int32_t *)malloc(sizeof(int32_t) * 4 * (size_t)ncells);
        int32_t *cand_q = (int32_t *)malloc(sizeof(int32_t) * 4 * (size_t)ncells);
        int32_t *cand_k = (int32_t *)malloc(sizeof(int32_t) * 4 * (size_t)ncells);
        if (!w.num || !w.den || !w.cnt || !Jloc || !cloc || !seen || !stamp || !cand_p || !cand_q || !cand_k) {
#pragma omp atomic write
            fail = 1;
        } else {
#pragma omp for schedule(dynamic, 1)
            for (int i = 0; i < ndirs; ++i) {
                orc_dir_t d;
                make_dir(&dirs[3 * i], &d);
                const int Na = w.dims[d.a], Nb = w.dims[d.b], Nc = w.dims[d.c];
                int pmin, qmin;
                lattice_range(w.dims, &d, &pmin, &qmin);
                w.pmin = pmin; w.qmin = qmin; w.np = Nb - pmin; w.nq = Nc - qmin;
                /* candidate rays: those whose entry cell in the sampled cell's slab is the cell itself or
                   its (-1,0), (0,-1), (-1,-1) neighbour (a ray's footprint in a slab is a 2x2 block).
                   A ray may be a candidate of several sampled cells; it is traced once per direction, from
                   its start to the slab of the last sampled cell it can touch (nothing downstream of that
                   slab is sampled): seen[(q - qmin) * np + (p - pmin)] = position + 1 in the candidate
                   list of this direction, stamp[] = index + 1 of the direction that wrote it. */
                int ncand = 0;
                for (int s = 0; s < ncells; ++s) {
                    int idx[3] = {cells[3 * s], cells[3 * s + 1], cells[3 * s + 2]};
                    int k = d.refl[d.a] ? Na - 1 - idx[d.a] : idx[d.a];
                    int j = d.refl[d.b] ? Nb - 1 - idx[d.b] : idx[d.b];
                    int l = d.refl[d.c] ? Nc - 1 - idx[d.c] : idx[d.c];
                    /* entry cell of ray p in slab k is floor((p + 1/2) + k Mb / ONE) = p + floor((ONE/2 + k Mb)/ONE) */
                    int64_t sb = (ORC_ONE / 2 + (int64_t)k * d.Mb) >> ORC_F;
                    int64_t sc = (ORC_ONE / 2 + (int64_t)k * d.Mc) >> ORC_F;
                    for (int dq = 0; dq <= 1; ++dq)
                        for (int dp = 0; dp <= 1; ++dp) {
                            int64_t p = j - dp - sb, q = l - dq - sc;
                            if (p < pmin || q < qmin) continue;         /* not a lattice ray: it never meets the box (O3) */
                            const size_t at = (size_t)(q - qmin) * w.np + (size_t)(p - pmin);
                            if (stamp[at] == i + 1) {
                                if (cand_k[seen[at]] < k) cand_k[seen[at]] = k;
                                continue;
                            }
                            stamp[at] = i + 1; seen[at] = ncand;
                            cand_p[ncand] = (int32_t)p; cand_q[ncand] = (int32_t)q; cand_k[ncand] = k;
                            ++ncand;
                        }
                }
                for (int r = 0; r < ncand; ++r) {
                    w.kstop = cand_k[r] + 1;
                    trace_ray(&w, &d, cand_p[r], cand_q[r]);
                }
                const double wgt = 1.0 / (double)ndirs;
                for (int s = 0; s < ncells; ++s) {
                    size_t cidx = (size_t)cells[3 * s + 2] * ny * nx + (size_t)cells[3 * s + 1] * nx + cells[3 * s];
                    double dn = w.den[cidx];
                    if (dn > 0.0)
                        for (int bin = 0; bin < nbins; ++bin)
                            Jloc[(size_t)bin * ncells + s] += wgt * w.num[(size_t)bin * ncell + cidx] / dn;
                    cloc[s] += w.cnt[cidx];
                    for (int bin = 0; bin < nbins; ++bin) w.num[(size_t)bin * ncell + cidx] = 0.0;
                    w.den[cidx] = 0.0; w.cnt[cidx] = 0;
                }
            }
#pragma omp critical
            {
                for (size_t o = 0; o < (size_t)ncells * nbins; ++o) Jin_out[o] += Jloc[o];
                if (cnt_out) for (int s = 0; s < ncells; ++s) cnt_out[s] += cloc[s];
            }
        }
        free(w.num); free(w.den); free(w.cnt); free(Jloc); free(cloc); free(seen); free(stamp); free(cand_p); free(cand_q); free(cand_k);
    }
    if (!fail && J_out)
        for (int bin = 0; bin < nbins; ++bin)
            for (int s = 0; s < ncells; ++s) {
                size_t cidx = (size_t)cells[3 * s + 2] * ny * nx + (size_t)cells[3 * s + 1] * nx + cells[3 * s];
                J_out[(size_t)bin * ncells + s] = Jin_out[(size_t)bin * ncells + s] + (double)S[(size_t)bin * ncell + cidx];
            }
    free(slot);
    return fail ? -2 : 0;
}

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ================================================================================================
 * Point radiation sources (section 2.1; Appendix 1) -- fp64.
 *
 * For every source alpha and every target cell one light-ray runs from the source to the centre of the
 * cell (Fig. 1) and on through the cell.  tau = sum of kappa*ds over the cells crossed
 * before the target cell (eq. 4's optical depth, up to the inner intersection r_in of Appendix 1),
 * dtau = kappa_cell * (r_out - r_in).  Photon-conserving absorption rate per unit volume of the shell
 * between r_in and r_out (eqs. A1-A3 divided by the shell volume; A5 is this divided by the species'
 * number density):
 *     Q[bin][cell] = sum_alpha  L[alpha][bin] * exp(-tau) * (1 - exp(-dtau)) / (4 pi/3 (r_out^3 - r_in^3))
 * Readings: source positions are given in units of 1/256 cell (integers), so
 * every decision of the traversal is exact integer arithmetic; a ray through an edge or corner steps all
 * the axes involved at once (zero-length pieces dropped, as A3); the source's own cell has r_in = 0.
 *   src_fix : int32 [nsrc][3] source positions in units of 1/256 cell width, inside the box
 *   lum     : fp64 [nsrc][nbins]
 *   Q       : fp64 [nbins][ncell] (may be NULL)
 *   tau_out, dtau_out, rin_out, rout_out : fp64 [ncell] for source `diag_src` and bin `diag_bin` (may be NULL)
 *   steps   : total number of positive-length segments marched (all sources, one bin)
 */
#define PS_FIX 256

typedef struct { int64_t num, den; } ps_rat_t;      /* den > 0 */
static int ps_less(ps_rat_t a, ps_rat_t b) { return (__int128)a.num * b.den < (__int128)b.num * a.den; }
static int ps_equal(ps_rat_t a, ps_rat_t b) { return (__int128)a.num * b.den == (__int128)b.num * a.den; }

int orc_point_sources(int nx, int ny, int nz, int nbins, const float *kappa, int nsrc, const int32_t *src_fix,
                      const double *lum, double cell_width, double *Q, int diag_src, int diag_bin,
                      double *tau_out, double *dtau_out, double *rin_out, double *rout_out,
                      unsigned long long *steps, int nthreads)
{
    if (nx < 1 || ny < 1 || nz < 1 || nbins < 1 || nbins > 16 || !kappa || nsrc < 1 || !src_fix || !lum) return -1;
    const int dims[3] = {nx, ny, nz};
    for (int a = 0; a < nsrc; ++a)
        for (int i = 0; i < 3; ++i)
            if (src_fix[3 * a + i] < 0 || src_fix[3 * a + i] > dims[i] * PS_FIX) return -1;
    const size_t ncell = (size_t)nx * ny * nz;
    const size_t stride[3] = {1, (size_t)nx, (size_t)nx * ny};
    if (Q) memset(Q, 0, sizeof(double) * ncell * nbins);
    unsigned long long nstep = 0;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
#pragma omp parallel for schedule(dynamic, 64) reduction(+ : nstep)
    for (long long cidx = 0; cidx < (long long)ncell; ++cidx) {
        int tgt[3] = {(int)(cidx % nx), (int)((cidx / nx) % ny), (int)(cidx / ((long long)nx * ny))};
        for (int a = 0; a < nsrc; ++a) {
            int64_t s[3], d[3];                                   /* source, and source -> cell centre, in 1/256 cells */
            int cur[3], stp[3];
            double len2 = 0.0;
            for (int i = 0; i < 3; ++i) {
                s[i] = src_fix[3 * a + i];
                d[i] = ((int64_t)tgt[i] * PS_FIX + PS_FIX / 2) - s[i];
                stp[i] = d[i] > 0 ? 1 : (d[i] < 0 ? -1 : 0);
                len2 += (double)d[i] * (double)d[i];
            }
            const double len = sqrt(len2) / PS_FIX * cell_width;  /* |centre - source| */
            /* cell containing the source, as seen from the ray: a source on a cell boundary belongs to the
               cell the ray moves into (d[i] == 0 cannot happen on a boundary: centres are half-integers) */
            for (int i = 0; i < 3; ++i) {
                int64_t c = s[i] / PS_FIX;
                if (s[i] % PS_FIX == 0 && stp[i] < 0) c -= 1;
                cur[i] = (int)c;
            }
            double tau[16];
            for (int b = 0; b < nbins; ++b) tau[b] = 0.0;
            ps_rat_t u0 = {0, 1};                                  /* ray parameter: 0 at the source, 1 at the centre */
            double r_in = 0.0, r_out = 0.0;
            for (;;) {
                /* next boundary crossing per axis: u_i = (plane_i - s_i) / d_i */
                ps_rat_t un = {1, 0};                              /* +infinity */
                int have = 0;
                ps_rat_t ui[3];
                for (int i = 0; i < 3; ++i) {
                    if (stp[i] == 0) continue;
                    int64_t plane = (int64_t)(cur[i] + (stp[i] > 0 ? 1 : 0)) * PS_FIX;
                    ui[i].num = (plane - s[i]) * stp[i];
                    ui[i].den = d[i] * stp[i];
                    if (!have || ps_less(ui[i], un)) { un = ui[i]; have = 1; }
                }
                const int is_target = (cur[0] == tgt[0] && cur[1] == tgt[1] && cur[2] == tgt[2]);
                const double t0 = (double)u0.num / (double)u0.den * len;
                const double t1 = have ? (double)un.num / (double)un.den * len : t0;
                const size_t cc = cur[0] * stride[0] + cur[1] * stride[1] + cur[2] * stride[2];
                if (is_target) {
                    r_in = t0; r_out = t1; nstep += 1;
                    if (!have) { r_in = 0.0; r_out = 0.5 * cell_width; }   /* source at this cell's centre: inscribed sphere */
                    break;
                }
                const double ds = t1 - t0;
                if (ds > 0.0) {
                    for (int b = 0; b < nbins; ++b) tau[b] += (double)kappa[(size_t)b * ncell + cc] * ds;
                    nstep += 1;
                }
                for (int i = 0; i < 3; ++i)                        /* all axes that cross at u_next step together */
                    if (stp[i] != 0 && ps_equal(ui[i], un)) cur[i] += stp[i];
                u0 = un;
            }
            const double vol = 4.0 * 3.14159265358979323846 / 3.0 * (r_out * r_out * r_out - r_in * r_in * r_in);
            for (int b = 0; b < nbins; ++b) {
                const double dtau = (double)kappa[(size_t)b * ncell + cidx] * (r_out - r_in);
                if (Q) Q[(size_t)b * ncell + cidx] += lum[(size_t)a * nbins + b] * exp(-tau[b]) * (-expm1(-dtau)) / vol;   /* A3 / V_shell */
                if (a == diag_src && b == diag_bin) {
                    if (tau_out) tau_out[cidx] = tau[b];
                    if (dtau_out) dtau_out[cidx] = dtau;
                }
            }
            if (a == diag_src) {
                if (rin_out) rin_out[cidx] = r_in;
                if (rout_out) rout_out[cidx] = r_out;
            }
        }
    }
    if (steps) *steps = nstep;
    return 0;
}
