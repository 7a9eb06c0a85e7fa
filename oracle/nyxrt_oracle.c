/*
 * nyxrt_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * A plain, slow, single-threaded fp64 CPU statement of ONE adaptive ray-tracing step on a
 * uniform coarse grid, written from the paper (arxiv 2512.12466, text at
 * /root/reference/PAPER.md; "PAPER.md:<line>" below) with the readings R1..R39 recorded in
 * DESIGN.md ("Readings").  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference leg may load this file.  It shares no code, header, table or helper with the
 * CUDA library under paper_2512_12466_b200/csrc and neither includes the other.
 *
 * Order of the step ("Ray tracing loop", 311 "collect ... duplicates ...
 * sorted", 313-333 + Alg. 3 at 343-391 "source merging"):
 *   orc_prepare_sources   dedup same-cell sources, sort
 *   orc_bubble_radius     MAX_RADIUS of Alg. 3
 *   orc_merge             MERGE_SOURCES of Alg. 3
 *   orc_trace             spawn 12 HEALPix rays per source; march / deposit / filter / split
 *                         depth-first until no ray is left                  (PAPER.md:111-128,
 *                         152-199, 83-95 Eq. 1-2, 211-249 Eq. 5-8)
 *   orc_step              the four above in order.
 *   orc_timestep          orc_step inside the iterative RT <-> ODE solve with the time-averaged update
 *                         of Eq. 3 (orc_ode_cell)                          ([23])
 *
 * Traversal is depth-first and recursive (a split recurses into the four children), which is
 * structurally unlike the CUDA library's pooled breadth-first loop.
 *
 * Floating point: everything is IEEE binary64; compile with -O2 -ffp-contract=off and no
 * fast-math.  fma() is used only where DESIGN.md writes fma.  Expressions that steer control
 * flow ("DEC" in DESIGN.md) are written exactly in the association DESIGN.md gives.
 *
 * Pins (tests/test_oracle_*.py, all -m "not gpu"): HEALPix ring heights / populations and the
 * inverse map ang->pix (Gorski et al. 2005, PAPER.md:613 ref [63]); slab-method exit distance and
 * fine-sampled cell lists for the DDA; tau closed form (Eq. 2); photon budget; thin-limit
 * Gamma = sigma Ndot exp(-tau) / (4 pi R^2) (Eq. 1 with V_shell); Stroemgren I-front, Eq. 10-11
 * with Table 1 Test A; Eq. 5-8 special cases; split radii from Eq. 4;
 * brute-force O(N^2)+DFS merge.  Parity UNPINNED by the paper (no printed values): the bubble
 * sample pattern and the merge defaults (PAPER.md:315-333 leave them to the user), the
 * figures 3, 4, 8c, and the reading of footnote 3 taken for thin segments -- the
 * thin table evaluated at the segment's midpoint and the neighbour's share taken from it, R41-R42:
 * T itself, the thin form's accuracy and the budget are pinned, the choice of reading is not.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORC_OK        0
#define ORC_EINVAL   -1
#define ORC_ENOMEM   -3
#define ORC_EOVERFLOW -5

#define ORC_MAXLEV 16

typedef struct {
    int32_t nx, ny, nz;
    int32_t field_dtype;      /* 0 = double fields, 1 = float fields (converted on load, exact) */
    double  dx_cm;            /* cubic cell width */
    double  box_lo[3];        /* low corner of cell (0,0,0), in position units */
    double  pos_unit_cm;      /* cm per position unit */
    int32_t periodic;         /* 0: rays leaving the box are removed (R20); 1: periodic box */
    int32_t pad_;
} orc_grid;

typedef struct {
    double  sigma_cm2;        /* monochromatic cross-section                                  */
    double  n_min_ray;        /* N_min^ray of Eq. 4                         */
    double  tau_max;          /* RAY_FLTR threshold                             */
    double  n_th;             /* Eq. 7-8 threshold                          */
    double  e_excess_erg;     /* heating per photo-ionisation (reading H1)                     */
    double  automerge_xmean;
    double  delta_r, r_max, f_ov, x_th, f_req, eps;   /* Alg. 3             */
    int32_t level_max;        /* l_max of RAY_FLTR                                             */
    int32_t geom_mode;        /* 0 none, 1 Eq.5 only, 2 Eq.5-6, 3 Eq.7-8, 4 squared [59]       */
    int32_t merge;            /* 0 off, 1 on, 2 automerge                                      */
    int32_t n_min_samples;    /* N_min of PAPER.md:317                                         */
    int32_t samp_level;       /* HEALPix level of the shell sample pattern (reading R6)        */
    int32_t pad_;
} orc_params;

typedef struct {
    uint64_t spawned[ORC_MAXLEV], split[ORC_MAXLEV], killed_tau[ORC_MAXLEV], exited[ORC_MAXLEV],
             killed_lmax[ORC_MAXLEV];
    uint64_t segments, zero_len_segments;
    uint64_t neighbour_deposits;   /* segments whose nearest neighbour received a share (Eq. 6 / 8) */
    uint64_t n_src_in, n_src_dedup, n_src_merged;
    double   photons_emitted, photons_absorbed, photons_escaped, photons_residual, photons_lost;
} orc_stats;

/* one record per ray-cell segment, optional (tests only) */
typedef struct {
    int32_t src, level;
    int64_t pix;
    int32_t cell[3];          /* absolute cell of the segment */
    int32_t nb_face;          /* 0..5 = x-,x+,y-,y+,z-,z+ if the neighbour got a share, else -1 */
    double  s0, ds, dtau, dN, fc, d_edge, l_pix;
} orc_seg;

/* ------------------------------------------------------------------------------------------ */
/* fields                                                                                      */

static inline double fld(const void *p, int dtype, int64_t i) {
    return dtype ? (double)((const float *)p)[i] : ((const double *)p)[i];
}

/* ------------------------------------------------------------------------------------------ */
/* O2: HEALPix nested pixel centre -> unit vector, "DIR-SPEC".                      */
/* Pixel geometry: Gorski et al. 2005 (PAPER.md:613 [63]); nested children of p are 4p..4p+3    */
/* ("splits into four HEALPix subpixels").                                        */

static double sin_poly(double x) {          /* Taylor through x^17, Horner, one fma per step  */
    double u = x * x, f = 1.0, c[9];
    int n = 1;
    for (int k = 0; k < 9; ++k) {           /* c[k] = (-1)^k / (2k+1)!  (division is exact-rounded) */
        c[k] = ((k & 1) ? -1.0 : 1.0) / f;
        f = f * (double)(n + 1) * (double)(n + 2);
        n += 2;
    }
    double p = c[8];
    for (int k = 7; k >= 0; --k) p = fma(p, u, c[k]);
    return x * p;
}

static double cos_poly(double x) {          /* Taylor through x^18 */
    double u = x * x, f = 1.0, c[10];
    int n = 0;
    for (int k = 0; k < 10; ++k) {          /* c[k] = (-1)^k / (2k)! */
        c[k] = ((k & 1) ? -1.0 : 1.0) / f;
        f = f * (double)(n + 1) * (double)(n + 2);
        n += 2;
    }
    double q = c[9];
    for (int k = 8; k >= 0; --k) q = fma(q, u, c[k]);
    return q;
}

int orc_pix2dir(int level, int64_t pix, double *d) {
    if (level < 0 || level > 14) return ORC_EINVAL;
    int64_t ns = (int64_t)1 << level, npf = ns * ns;
    if (pix < 0 || pix >= 12 * npf) return ORC_EINVAL;
    int64_t f = pix / npf, pf = pix % npf;
    int64_t row = f / 4;
    int64_t ix = 0, iy = 0;
    for (int b = 0; b < level; ++b) {
        ix |= ((pf >> (2 * b)) & 1) << b;
        iy |= ((pf >> (2 * b + 1)) & 1) << b;
    }
    int64_t jr = (row + 2) * ns - ix - iy - 1;        /* ring, 1-based from the north pole */
    int64_t nr, k;
    double z, st;
    if (jr < ns) {                                    /* north cap */
        nr = jr; k = 0;
        double t = (double)(nr * nr) / (double)(3 * ns * ns);
        z = 1.0 - t;
        st = sqrt(t * (2.0 - t));
    } else if (jr > 3 * ns) {                         /* south cap */
        nr = 4 * ns - jr; k = 0;
        double t = (double)(nr * nr) / (double)(3 * ns * ns);
        z = t - 1.0;
        st = sqrt(t * (2.0 - t));
    } else {                                          /* equatorial belt */
        nr = ns; k = (jr - ns) & 1;
        z = ((double)(2 * ns - jr) * 2.0) / (double)(3 * ns);
        st = sqrt((1.0 - z) * (1.0 + z));
    }
    int64_t jf = 2 * (f % 4) + (row == 1 ? 0 : 1);
    int64_t jp = (jf * nr + ix - iy + 1 + k) / 2;
    if (jp > 4 * nr) jp -= 4 * nr;
    if (jp < 1) jp += 4 * nr;
    int64_t m = 2 * jp - k - 1;                       /* phi = (pi/4) m / nr, 0 <= m < 8 nr */
    int64_t q = m / nr, rem = m % nr;
    int64_t num = (q & 1) ? (nr - rem) : rem;
    const double PI_4 = 0x1.921fb54442d18p-1;
    double alpha = (PI_4 * (double)num) / (double)nr;
    double c = cos_poly(alpha), s = sin_poly(alpha);
    if (num == nr) c = s = 0x1.6a09e667f3bcdp-1;       /* phi on a diagonal: cos = sin = sqrt(1/2) exactly alike */
    double cp, sp;
    switch ((int)q) {
        case 0: cp = c;  sp = s;  break;
        case 1: cp = s;  sp = c;  break;
        case 2: cp = -s; sp = c;  break;
        case 3: cp = -c; sp = s;  break;
        case 4: cp = -c; sp = -s; break;
        case 5: cp = -s; sp = -c; break;
        case 6: cp = s;  sp = -c; break;
        default: cp = c; sp = -s; break;
    }
    d[0] = st * cp;
    d[1] = st * sp;
    d[2] = z;
    return ORC_OK;
}

/* ------------------------------------------------------------------------------------------ */
/* O1: source preparation ("duplicates (sources assigned to the same grid cell)     */
/* are identified and merged by summing their fluxes. The resulting deduplicated list is then    */
/* sorted"; "S has integer coords").                                               */

typedef struct { int64_t key; int64_t idx; } keyidx;

static int cmp_keyidx(const void *a, const void *b) {
    const keyidx *x = a, *y = b;
    if (x->key != y->key) return x->key < y->key ? -1 : 1;
    return x->idx < y->idx ? -1 : (x->idx > y->idx);
}

/* out_cell: [n][3] int32, out_L: [n]; returns count in *n_out (<= n) */
int orc_prepare_sources(const orc_grid *g, int64_t n, const double *pos, const double *L,
                        int32_t *out_cell, double *out_L, int64_t *n_out) {
    *n_out = 0;
    if (n < 0) return ORC_EINVAL;
    if (n == 0) return ORC_OK;
    keyidx *ki = malloc((size_t)n * sizeof *ki);
    if (!ki) return ORC_ENOMEM;
    for (int64_t a = 0; a < n; ++a) {
        int64_t c[3];
        int32_t dim[3] = { g->nx, g->ny, g->nz };
        if (!(L[a] >= 0.0) || isinf(L[a])) { free(ki); return ORC_EINVAL; }
        for (int ax = 0; ax < 3; ++ax) {
            double u = (pos[3 * a + ax] - g->box_lo[ax]) * g->pos_unit_cm / g->dx_cm;
            if (!(u >= 0.0) || !(u < (double)dim[ax])) { free(ki); return ORC_EINVAL; }
            c[ax] = (int64_t)floor(u);
            if (c[ax] >= dim[ax]) { free(ki); return ORC_EINVAL; }
        }
        ki[a].key = (c[2] * g->ny + c[1]) * (int64_t)g->nx + c[0];
        ki[a].idx = a;
    }
    qsort(ki, (size_t)n, sizeof *ki, cmp_keyidx);       /* (key, input index): stable by construction */
    int64_t m = 0;
    for (int64_t a = 0; a < n;) {
        int64_t b = a;
        double sum = 0.0;
        while (b < n && ki[b].key == ki[a].key) { sum = sum + L[ki[b].idx]; ++b; }  /* input order */
        int64_t key = ki[a].key;
        out_cell[3 * m + 0] = (int32_t)(key % g->nx);
        out_cell[3 * m + 1] = (int32_t)((key / g->nx) % g->ny);
        out_cell[3 * m + 2] = (int32_t)(key / ((int64_t)g->nx * g->ny));
        out_L[m] = sum;
        ++m;
        a = b;
    }
    free(ki);
    *n_out = m;
    return ORC_OK;
}

/* ------------------------------------------------------------------------------------------ */
/* M1-M4: MAX_RADIUS (Alg. 3; text 313-319).                                   */

static int in_box(const orc_grid *g, int64_t i, int64_t j, int64_t k) {
    return i >= 0 && i < g->nx && j >= 0 && j < g->ny && k >= 0 && k < g->nz;
}

static int64_t lin(const orc_grid *g, int64_t i, int64_t j, int64_t k) {
    return (k * g->ny + j) * (int64_t)g->nx + i;
}

/* periodic box ("rays wrap around the box"): index into [0, n) */
static int64_t wrap(int64_t i, int64_t n) {
    i %= n;
    return i < 0 ? i + n : i;
}

/* minimum-image difference of two cell coordinates ("minimum-image convention"): the
   representative of a - b (mod n) in [-n/2, n/2); for even n the tie n/2 maps to -n/2 (reading R31) */
static int64_t minimg(int64_t d, int64_t n) {
    d = wrap(d, n);
    return (2 * d >= n) ? d - n : d;
}

int orc_bubble_radius(const orc_grid *g, const orc_params *p, const void *xHI, int64_t n,
                      const int32_t *cell, double *r_out) {
    if (p->samp_level < 0 || p->samp_level > 8 || !(p->delta_r > 0.0)) return ORC_EINVAL;
    int64_t ns = (int64_t)12 << (2 * p->samp_level);
    double *dir = malloc((size_t)ns * 3 * sizeof *dir);
    if (!dir) return ORC_ENOMEM;
    for (int64_t q = 0; q < ns; ++q) orc_pix2dir(p->samp_level, q, dir + 3 * q);
    for (int64_t a = 0; a < n; ++a) {
        const int32_t *c = cell + 3 * a;
        double x0 = 1.0 - fld(xHI, g->field_dtype, lin(g, c[0], c[1], c[2]));  /* ionised fraction */
        if (x0 < p->x_th) { r_out[a] = 0.0; continue; }
        double r = p->delta_r, res = -1.0;
        while (r <= p->r_max) {
            int64_t ntot = 0, nion = 0;
            for (int64_t q = 0; q < ns; ++q) {
                int64_t i = c[0] + (int64_t)floor(fma(r, dir[3 * q + 0], 0.5));
                int64_t j = c[1] + (int64_t)floor(fma(r, dir[3 * q + 1], 0.5));
                int64_t k = c[2] + (int64_t)floor(fma(r, dir[3 * q + 2], 0.5));
                if (g->periodic) { i = wrap(i, g->nx); j = wrap(j, g->ny); k = wrap(k, g->nz); }
                else if (!in_box(g, i, j, k)) continue;                       /* "checked" samples */
                ++ntot;
                double x = 1.0 - fld(xHI, g->field_dtype, lin(g, i, j, k));
                if (x >= p->x_th) ++nion;
            }
            int pass;
            if (ntot == 0) pass = 0;                                          /* reading R7 */
            else if (ntot < p->n_min_samples) pass = (nion == ntot);
            else pass = ((double)nion >= p->f_req * (double)ntot);
            if (!pass) { res = r - p->delta_r; break; }
            r = r + p->delta_r;
        }
        r_out[a] = (res >= 0.0) ? res : p->r_max;
    }
    free(dir);
    return ORC_OK;
}

/* ------------------------------------------------------------------------------------------ */
/* M5-M8: MERGE_SOURCES (Alg. 3; text 321-333).  All pairs, union-find.        */

static int64_t uf_find(int64_t *par, int64_t a) {
    while (par[a] != a) { par[a] = par[par[a]]; a = par[a]; }
    return a;
}

typedef struct { int64_t key; int32_t c[3]; double L, r; } msrc;

static int cmp_msrc(const void *a, const void *b) {
    const msrc *x = a, *y = b;
    return x->key < y->key ? -1 : (x->key > y->key);
}

int orc_merge(const orc_grid *g, const orc_params *p, int64_t n, const int32_t *cell,
              const double *L, const double *r, int32_t *out_cell, double *out_L, double *out_r,
              int64_t *n_out) {
    *n_out = 0;
    if (n <= 0) return n < 0 ? ORC_EINVAL : ORC_OK;
    int64_t *par = malloc((size_t)n * sizeof *par);
    int64_t *minm = malloc((size_t)n * sizeof *minm);
    msrc *out = malloc((size_t)n * sizeof *out);
    if (!par || !minm || !out) { free(par); free(minm); free(out); return ORC_ENOMEM; }
    for (int64_t a = 0; a < n; ++a) par[a] = a;
    for (int64_t a = 0; a < n; ++a) {
        if (!(r[a] > 0.0)) continue;
        for (int64_t b = a + 1; b < n; ++b) {
            if (!(r[b] > 0.0)) continue;
            int64_t dx = (int64_t)cell[3 * a] - cell[3 * b], dy = (int64_t)cell[3 * a + 1] - cell[3 * b + 1],
                    dz = (int64_t)cell[3 * a + 2] - cell[3 * b + 2];
            if (g->periodic) { dx = minimg(dx, g->nx); dy = minimg(dy, g->ny); dz = minimg(dz, g->nz); }
            int64_t d2 = dx * dx + dy * dy + dz * dz;
            double rs = p->f_ov * (r[a] + r[b]);
            if ((double)d2 <= rs * rs + p->eps) {
                int64_t ra = uf_find(par, a), rb = uf_find(par, b);
                if (ra != rb) { if (ra < rb) par[rb] = ra; else par[ra] = rb; }
            }
        }
    }
    /* smallest member of each component (roots are already the smallest by construction, but do
       not rely on it) */
    for (int64_t a = 0; a < n; ++a) minm[a] = n;
    for (int64_t a = 0; a < n; ++a) { int64_t ra = uf_find(par, a); if (a < minm[ra]) minm[ra] = a; }
    int64_t m = 0;
    for (int64_t a = 0; a < n; ++a) {               /* groups in order of their smallest member */
        int64_t ra = uf_find(par, a);
        if (minm[ra] != a) continue;
        int64_t cnt = 0;
        for (int64_t b = a; b < n; ++b) if (uf_find(par, b) == ra) ++cnt;
        msrc M;
        if (cnt == 1) {
            M.c[0] = cell[3 * a]; M.c[1] = cell[3 * a + 1]; M.c[2] = cell[3 * a + 2];
            M.L = L[a]; M.r = r[a];
        } else {
            const int64_t nn[3] = { g->nx, g->ny, g->nz };
            double F = 0.0, R = 0.0, num[3] = { 0.0, 0.0, 0.0 };
            for (int64_t b = a; b < n; ++b) {                                 /* member order */
                if (uf_find(par, b) != ra) continue;
                F = F + L[b];
                if (r[b] > R) R = r[b];
                for (int ax = 0; ax < 3; ++ax) {
                    /* periodic: x'_m = x_ref + minimg(x_m - x_ref), reference = first member */
                    int64_t x = cell[3 * b + ax];
                    if (g->periodic) x = cell[3 * a + ax] + minimg(x - cell[3 * a + ax], nn[ax]);
                    num[ax] = num[ax] + L[b] * (double)x;
                }
            }
            int64_t rc[3];
            for (int ax = 0; ax < 3; ++ax) {
                rc[ax] = (int64_t)floor(num[ax] / F + 0.5);                   /* R9 */
                if (g->periodic) rc[ax] = wrap(rc[ax], nn[ax]);               /* "wrapped back into the box" */
            }
            int64_t best = -1, bestd = 0;
            for (int64_t b = a; b < n; ++b) {                                 /* snap */
                if (uf_find(par, b) != ra) continue;
                int64_t dx = cell[3 * b] - rc[0], dy = cell[3 * b + 1] - rc[1], dz = cell[3 * b + 2] - rc[2];
                if (g->periodic) { dx = minimg(dx, g->nx); dy = minimg(dy, g->ny); dz = minimg(dz, g->nz); }
                int64_t d2 = dx * dx + dy * dy + dz * dz;
                if (best < 0 || d2 < bestd) { best = b; bestd = d2; }         /* first minimum, R10 */
            }
            M.c[0] = cell[3 * best]; M.c[1] = cell[3 * best + 1]; M.c[2] = cell[3 * best + 2];
            M.L = F; M.r = R;
        }
        M.key = lin(g, M.c[0], M.c[1], M.c[2]);
        out[m++] = M;
    }
    qsort(out, (size_t)m, sizeof *out, cmp_msrc);                             /* PAPER.md:388; keys unique */
    for (int64_t a = 0; a < m; ++a) {
        out_cell[3 * a] = out[a].c[0]; out_cell[3 * a + 1] = out[a].c[1]; out_cell[3 * a + 2] = out[a].c[2];
        out_L[a] = out[a].L; out_r[a] = out[a].r;
    }
    *n_out = m;
    free(par); free(minm); free(out);
    return ORC_OK;
}

/* ------------------------------------------------------------------------------------------ */
/* O3-O7: the ray loop.                                                                          */

/* ------------------------------------------------------------------------------------------ */
/* S1-S3: frequency-integrated flux (Sec. 2.2): "the solution to Eq. 1 can be      */
/* precomputed as a function of tau_0 (optical depth at the ionization threshold frequency). A     */
/* lookup table allows us to sidestep the need for per-ray frequency bins".  With sigma_nu =        */
/* sigma_0 (nu/nu_0)^-3 (R37) and a photon-number spectrum phi(nu), int phi = 1, the photons a ray  */
/* of share w loses between tau_0 = a and b are w [Q(b) - Q(a)],                                    */
/*     Q(tau_0) = int phi(nu) (1 - exp(-tau_0 (nu/nu_0)^-3)) dnu          (Eq. 1's numerator),      */
/* which telescopes along the ray (photon conservation).  Q is tabulated on nodes fixed by the      */
/* binary representation of tau_0 (R38): 2^m nodes per octave, linear in tau_0 inside an octave,    */
/* from 2^e_lo to 2^e_hi; linear from 0 below 2^e_lo; constant above 2^e_hi.                        */

static struct { int on, e_lo, e_hi, m; int64_t n; double *q; double *t; double tau_thin; } g_lut;

int64_t orc_spectrum_nodes(int e_lo, int e_hi, int m) { return (((int64_t)(e_hi - e_lo)) << m) + 1; }

/* tau_0 of node k */
double orc_spectrum_node_tau(int e_lo, int m, int64_t k) {
    int64_t oct = k >> m, sub = k & (((int64_t)1 << m) - 1);
    return ldexp(1.0 + (double)sub / (double)((int64_t)1 << m), e_lo + (int)oct);
}

int orc_set_spectrum(int e_lo, int e_hi, int m, const double *q, int64_t n) {
    if (q) {                                                            /* a rejected call leaves both tables as they were */
        if (e_lo < -1000 || e_hi > 1000 || e_hi <= e_lo || m < 0 || m > 20 || n != orc_spectrum_nodes(e_lo, e_hi, m))
            return ORC_EINVAL;
    }
    double *copy = NULL;
    if (q) {
        copy = malloc((size_t)n * sizeof *q);
        if (!copy) return ORC_ENOMEM;
        memcpy(copy, q, (size_t)n * sizeof *q);
    }
    free(g_lut.q);
    free(g_lut.t);                                                      /* a new Q table drops the thin table */
    memset(&g_lut, 0, sizeof g_lut);
    if (!q) return ORC_OK;                                              /* back to monochromatic */
    g_lut.q = copy;
    g_lut.on = 1; g_lut.e_lo = e_lo; g_lut.e_hi = e_hi; g_lut.m = m; g_lut.n = n;
    return ORC_OK;
}

/* S2: table lookup (R38) */
double orc_spectrum_q(double tau) {
    if (!(tau > 0.0)) return 0.0;
    if (tau < ldexp(1.0, g_lut.e_lo)) return g_lut.q[0] * ldexp(tau, -g_lut.e_lo);
    if (tau >= ldexp(1.0, g_lut.e_hi)) return g_lut.q[g_lut.n - 1];
    uint64_t bits;
    memcpy(&bits, &tau, sizeof bits);
    const int fb = 52 - g_lut.m;                                        /* mantissa bits below the node */
    int64_t k = (int64_t)(bits >> fb) - ((int64_t)(g_lut.e_lo + 1023) << g_lut.m);
    double frac = ldexp((double)(bits & (((uint64_t)1 << fb) - 1)), -fb);
    return fma(frac, g_lut.q[k + 1] - g_lut.q[k], g_lut.q[k]);
}

/* S4: the separate table for the optically thin case (PAPER.md:267 footnote 3: "the approach of C2-Ray, which
   takes the limit as n_H -> 0 to compute a separate LUT for the optically thin case"; with PAPER.md:95).  In the
   limit of a thin cell Eq. 1's factor (1 - exp(-dtau_nu)) -> dtau_nu = dtau_0 (nu/nu_0)^-3, so the share absorbed in
   the cell is dtau_0 T(tau_0) with
       T(tau_0) = int phi(nu) (nu/nu_0)^-3 exp(-tau_0 (nu/nu_0)^-3) dnu  =  dQ/dtau_0,
   tabulated on the nodes of Q and interpolated the same way (constant below the first node and above the last)
   [R40].  A segment with dtau_0 < tau_thin takes dtau_0 T(tau_0 + dtau_0 / 2) instead of Q(tau_0 + dtau_0) -
   Q(tau_0), the difference of two interpolants that cancels there [R41].  The two forms do not telescope into
   each other, so with the thin table set the photons a ray carries are counted down segment by segment instead of
   being read off Q(tau_0) [R42].  The neighbour's share (Eq. 6 / 8) is (1 - f_c) of whatever the segment absorbed,
   in photons: no quotient of absorber densities is formed, which is the part the footnote calls "not applicable". */
int orc_set_spectrum_thin(const double *t, int64_t n, double tau_thin) {
    double *copy = NULL;
    if (t) {                                                            /* a rejected call leaves the thin table in place */
        if (!g_lut.on || n != g_lut.n || !(tau_thin >= 0.0)) return ORC_EINVAL;
        copy = malloc((size_t)n * sizeof *t);
        if (!copy) return ORC_ENOMEM;
        memcpy(copy, t, (size_t)n * sizeof *t);
    }
    free(g_lut.t);
    g_lut.t = copy;
    g_lut.tau_thin = t ? tau_thin : 0.0;
    return ORC_OK;
}

double orc_spectrum_t(double tau) {
    if (!(tau >= ldexp(1.0, g_lut.e_lo))) return g_lut.t[0];
    if (tau >= ldexp(1.0, g_lut.e_hi)) return g_lut.t[g_lut.n - 1];
    uint64_t bits;
    memcpy(&bits, &tau, sizeof bits);
    const int fb = 52 - g_lut.m;
    int64_t k = (int64_t)(bits >> fb) - ((int64_t)(g_lut.e_lo + 1023) << g_lut.m);
    double frac = ldexp((double)(bits & (((uint64_t)1 << fb) - 1)), -fb);
    return fma(frac, g_lut.t[k + 1] - g_lut.t[k], g_lut.t[k]);
}

/* absorbed fraction of a ray's share between the source and optical depth tau; share absorbed in a
   segment from tau to tau + dtau (Eq. 1 with V_box) */
static double remaining_at(double tau) { return g_lut.on ? 1.0 - orc_spectrum_q(tau) : exp(-tau); }
static double absorbed_in(double tau, double dtau) {
    if (g_lut.on) {
        if (g_lut.t && dtau < g_lut.tau_thin) return dtau * orc_spectrum_t(tau + 0.5 * dtau);     /* R41 */
        return orc_spectrum_q(tau + dtau) - orc_spectrum_q(tau);
    }
    return exp(-tau) * (-expm1(-dtau));
}

/* S3: Q of a black body of temperature T_eff [K] (R39): phi(nu) ~ nu^2 / (exp(h nu / k T) - 1) above
   nu_0 (13.6 eV): with x = h nu / k T, x_0 = h nu_0 / k T,
       Q(tau) = int_{x0}^inf x^2/(e^x - 1) (1 - exp(-tau (x/x0)^-3)) dx / int_{x0}^inf x^2/(e^x - 1) dx,
   composite Simpson on u in [0, 1) with x = x0 + u/(1-u) (the integrand vanishes at u -> 1). */
static double bb_integral(double x0, double tau, int with_abs) {
    const int N = 20000;                                                /* even */
    double sum = 0.0;
    for (int i = 0; i < N; ++i) {                                       /* u = 1 excluded: integrand 0 */
        double u = (double)i / (double)N;
        double x = x0 + u / (1.0 - u);
        double jac = 1.0 / ((1.0 - u) * (1.0 - u));
        double f = x * x / expm1(x) * jac;
        if (with_abs == 1) { double r = x0 / x; f *= -expm1(-tau * r * r * r); }
        if (with_abs == 2) { double r = x0 / x; f *= (r * r * r) * exp(-tau * r * r * r); }    /* thin table T */
        double wgt = (i == 0) ? 1.0 : ((i & 1) ? 4.0 : 2.0);
        sum += wgt * f;
    }
    return sum / (3.0 * (double)N);
}

int orc_blackbody_table(double t_eff_K, int e_lo, int e_hi, int m, double *q, int64_t n) {
    if (!(t_eff_K > 0.0) || n != orc_spectrum_nodes(e_lo, e_hi, m)) return ORC_EINVAL;
    const double x0 = 13.598434 * 1.602176634e-19 / (1.380649e-23 * t_eff_K);   /* h nu_0 / k T */
    const double norm = bb_integral(x0, 0.0, 0);
    for (int64_t k = 0; k < n; ++k) q[k] = bb_integral(x0, orc_spectrum_node_tau(e_lo, m, k), 1) / norm;
    return ORC_OK;
}

/* T = dQ/dtau_0 of the same black body on the same nodes (S4, R40) */
int orc_blackbody_thin_table(double t_eff_K, int e_lo, int e_hi, int m, double *t, int64_t n) {
    if (!(t_eff_K > 0.0) || n != orc_spectrum_nodes(e_lo, e_hi, m)) return ORC_EINVAL;
    const double x0 = 13.598434 * 1.602176634e-19 / (1.380649e-23 * t_eff_K);
    const double norm = bb_integral(x0, 0.0, 0);
    for (int64_t k = 0; k < n; ++k) t[k] = bb_integral(x0, orc_spectrum_node_tau(e_lo, m, k), 2) / norm;
    return ORC_OK;
}

typedef struct {
    const orc_grid *g;
    const orc_params *p;
    const void *nH, *xHI;
    double *gamma, *heat;
    orc_stats *st;
    orc_seg *log;
    int64_t log_cap, log_n;
    double r2_split[ORC_MAXLEV], K[ORC_MAXLEV];
    double sdx, V;
    double s_max;             /* periodic: sqrt(nx^2 + ny^2 + nz^2) cells = sqrt(3) L_box for a cube */
    long double absorbed, escaped, residual, lost;
    int32_t src_cell[3];
    int32_t src_id;
    double L_src;
} tracer;

/* carried: photons/s the ray holds at birth; used (and counted down) only when the thin table is set (R42) */
static void trace_ray(tracer *T, int level, int64_t pix, double s, double tau, double carried) {
    const orc_grid *g = T->g;
    const orc_params *p = T->p;
    orc_stats *st = T->st;
    const double L_ray = T->L_src / (12.0 * ldexp(1.0, 2 * level));   /* L shared evenly */
    const int count_down = g_lut.on && g_lut.t != NULL;
#define RAY_PHOTONS() (count_down ? carried : L_ray * remaining_at(tau))
    double d[3], inv[3], sx[3];
    int64_t o[3];
    orc_pix2dir(level, pix, d);
    st->spawned[level]++;
    /* O4: start-of-life cell in source-relative cell units (source at its cell centre, R3) */
    for (int a = 0; a < 3; ++a) {
        double q = fma(s, d[a], 0.5);
        double fl = floor(q);
        o[a] = (int64_t)fl;
        if (q == fl && d[a] < 0.0) o[a] -= 1;                          /* R12 */
        if (d[a] == 0.0) { inv[a] = 0.0; sx[a] = INFINITY; }
        else {
            inv[a] = 1.0 / d[a];
            sx[a] = ((double)(o[a] + (d[a] > 0.0 ? 1 : 0)) - 0.5) * inv[a];
        }
    }
    if (!g->periodic && !in_box(g, T->src_cell[0] + o[0], T->src_cell[1] + o[1], T->src_cell[2] + o[2])) {
        st->exited[level]++;
        T->escaped += (long double)RAY_PHOTONS();
        return;
    }
    for (;;) {
        /* 1. kill (RAY_FLTR tau test; per cell, R14) */
        if (tau >= p->tau_max) {
            st->killed_tau[level]++;
            T->residual += (long double)RAY_PHOTONS();
            return;
        }
        /* 2. l_max */
        if (level >= p->level_max) {
            st->killed_lmax[level]++;
            T->residual += (long double)RAY_PHOTONS();
            return;
        }
        /* 2b. periodic box: the ray ends once its travel distance is no longer below sqrt(3) L_box
           (RAY_FLTR); counted with the rays that left the system (reading R30) */
        if (g->periodic && !(s < T->s_max)) {
            st->exited[level]++;
            T->escaped += (long double)RAY_PHOTONS();
            return;
        }
        /* 3. split, Eq. 4: Omega_c/Omega(l) < N_min  <=>  s^2 > 3 4^l/(pi N_min) */
        if (s * s > T->r2_split[level]) {
            st->split[level]++;
            for (int k = 0; k < 4; ++k) trace_ray(T, level + 1, 4 * pix + k, s, tau, 0.25 * carried);
            return;
        }
        /* 4. one cell (Amanatides-Woo, PAPER.md:152 [76]) */
        int ax = 0;
        double s_exit = sx[0];
        if (sx[1] < s_exit) { s_exit = sx[1]; ax = 1; }
        if (sx[2] < s_exit) { s_exit = sx[2]; ax = 2; }                /* first minimum, R19 */
        double ds = s_exit - s;
        if (!(ds > 0.0)) ds = 0.0;
        if (ds > 0.0) {
            st->segments++;
            int64_t ci = T->src_cell[0] + o[0], cj = T->src_cell[1] + o[1], ck = T->src_cell[2] + o[2];
            if (g->periodic) { ci = wrap(ci, g->nx); cj = wrap(cj, g->ny); ck = wrap(ck, g->nz); }
            int64_t c = lin(g, ci, cj, ck);
            double nH_c = fld(T->nH, g->field_dtype, c);
            double a_c = nH_c * fld(T->xHI, g->field_dtype, c);        /* absorber density, PAPER.md:229 (R1) */
            double dtau = (a_c * T->sdx) * ds;                         /* Eq. 2 */
            double dN = L_ray * absorbed_in(tau, dtau);                /* Eq. 1 with V_box */
            if (dN > 0.0) {
                double fc = 1.0, d_edge = 0.0, l_pix = 0.0, a_n = 0.0;
                int face = -1;
                int64_t cn = -1;                                       /* neighbour that gets a share */
                if (p->geom_mode != 0) {
                    /* Sec. 2.6: D_edge = distance from the segment midpoint to the
                       nearest cell face (R21), L_pix = linear width of the HEALPix pixel there (R22). */
                    double s_m = s + 0.5 * ds;
                    double cand[6];
                    for (int a = 0; a < 3; ++a) {
                        double m = fma(s_m, d[a], 0.5) - (double)o[a];
                        if (m < 0.0) m = 0.0;
                        if (m > 1.0) m = 1.0;
                        cand[2 * a] = m;                               /* low face  */
                        cand[2 * a + 1] = 1.0 - m;                     /* high face */
                    }
                    face = 0; d_edge = cand[0];
                    for (int f = 1; f < 6; ++f) if (cand[f] < d_edge) { d_edge = cand[f]; face = f; }
                    l_pix = s_m * T->K[level];
                    if (d_edge < 0.5 * l_pix) {                        /* first condition of Eq. 5 / 7 */
                        if (p->geom_mode == 1) fc = 0.5 + d_edge / l_pix;            /* Eq. 5 alone */
                        else if (p->geom_mode == 4) { fc = 0.5 + d_edge / l_pix; fc = fc * fc; }  /* [59] */
                        else {                                         /* 2: Eq. 5-6; 3: Eq. 7-8 */
                            int64_t nb[3] = { ci, cj, ck };
                            nb[face >> 1] += (face & 1) ? 1 : -1;
                            if (g->periodic) { nb[0] = wrap(nb[0], g->nx); nb[1] = wrap(nb[1], g->ny); nb[2] = wrap(nb[2], g->nz); }
                            if (in_box(g, nb[0], nb[1], nb[2])) {      /* R23 */
                                int64_t q = lin(g, nb[0], nb[1], nb[2]);
                                double nH_n = fld(T->nH, g->field_dtype, q);
                                a_n = nH_n * fld(T->xHI, g->field_dtype, q);
                                int ok = a_n > 0.0;                    /* R24 */
                                if (p->geom_mode == 3 && !(nH_n >= p->n_th)) ok = 0;   /* Eq. 7-8 */
                                if (ok) { fc = 0.5 + d_edge / l_pix; cn = q; }
                            }
                        }
                    }
                }
                double gC = dN / (a_c * T->V);                         /* Gamma of Eq. 1 for this segment */
                T->gamma[c] += fc * gC;
                if (T->heat) T->heat[c] += p->e_excess_erg * fc * dN / T->V;       /* H1 */
                long double dep = (long double)(fc * dN);
                if (cn >= 0) {
                    st->neighbour_deposits++;
                    double fn = (1.0 - fc) * (a_c / a_n);              /* Eq. 6 / Eq. 8: f_c' */
                    T->gamma[cn] += fn * gC;
                    if (T->heat) T->heat[cn] += p->e_excess_erg * (1.0 - fc) * dN / T->V;
                    dep += (long double)((1.0 - fc) * dN);
                } else if (fc < 1.0) {
                    T->lost += (long double)((1.0 - fc) * dN);         /* modes 1, 4 */
                }
                T->absorbed += dep;
                if (T->log && T->log_n < T->log_cap) {
                    orc_seg *r = &T->log[T->log_n];
                    r->src = T->src_id; r->level = level; r->pix = pix;
                    r->cell[0] = (int32_t)ci; r->cell[1] = (int32_t)cj; r->cell[2] = (int32_t)ck;
                    r->nb_face = (cn >= 0) ? face : -1;
                    r->s0 = s; r->ds = ds; r->dtau = dtau; r->dN = dN; r->fc = fc;
                    r->d_edge = d_edge; r->l_pix = l_pix;
                }
                if (T->log) T->log_n++;
            } else if (T->log) {
                if (T->log_n < T->log_cap) {
                    orc_seg *r = &T->log[T->log_n];
                    memset(r, 0, sizeof *r);
                    r->src = T->src_id; r->level = level; r->pix = pix;
                    r->cell[0] = (int32_t)ci; r->cell[1] = (int32_t)cj; r->cell[2] = (int32_t)ck;
                    r->nb_face = -1; r->s0 = s; r->ds = ds; r->dtau = dtau; r->fc = 1.0;
                }
                T->log_n++;
            }
            tau = tau + dtau;
            carried = carried - dN;
        } else {
            st->zero_len_segments++;
        }
        s = s_exit;
        o[ax] += (d[ax] > 0.0) ? 1 : -1;
        sx[ax] = ((double)(o[ax] + (d[ax] > 0.0 ? 1 : 0)) - 0.5) * inv[ax];
        if (!g->periodic && !in_box(g, T->src_cell[0] + o[0], T->src_cell[1] + o[1], T->src_cell[2] + o[2])) {
            st->exited[level]++;                                        /* R20 */
            T->escaped += (long double)RAY_PHOTONS();
            return;
        }
    }
}
#undef RAY_PHOTONS

/* gamma, heat: [nz][ny][nx] double; heat may be NULL.  zero != 0: overwritten; zero == 0: the deposits are ADDED
   to what the grids hold and the counters to *st (Gamma is a sum over sources: a catalogue can be
   traced slice by slice, or by several processes whose grids are added afterwards).  log may be NULL.
   *log_n_out (may be NULL) receives the number of segments that WOULD have been logged. */
static int trace_catalogue(const orc_grid *g, const orc_params *p, const void *nH, const void *xHI,
                           int64_t n_cat, const int32_t *cell, const double *L, double *gamma, double *heat,
                           orc_stats *st, orc_seg *log, int64_t log_cap, int64_t *log_n_out, int zero) {
    if (p->level_max < 0 || p->level_max >= ORC_MAXLEV - 1 || !(p->n_min_ray > 0.0)) return ORC_EINVAL;
    if (p->geom_mode < 0 || p->geom_mode > 4) return ORC_EINVAL;
    int64_t ncell = (int64_t)g->nx * g->ny * g->nz;
    if (zero) {
        memset(gamma, 0, (size_t)ncell * sizeof *gamma);
        if (heat) memset(heat, 0, (size_t)ncell * sizeof *heat);
    }
    tracer T;
    memset(&T, 0, sizeof T);
    T.g = g; T.p = p; T.nH = nH; T.xHI = xHI; T.gamma = gamma; T.heat = heat; T.st = st;
    T.log = log; T.log_cap = log_cap; T.log_n = 0;
    const double PI = 0x1.921fb54442d18p+1;
    for (int l = 0; l < ORC_MAXLEV; ++l) {
        T.r2_split[l] = ldexp(3.0 / (PI * p->n_min_ray), 2 * l);       /* Eq. 4 */
        T.K[l] = ldexp(sqrt(PI / 3.0), -l);                            /* sqrt(Omega(l)), R22 */
    }
    T.sdx = p->sigma_cm2 * g->dx_cm;
    T.V = g->dx_cm * g->dx_cm * g->dx_cm;                              /* V_box = h^3 */
    T.s_max = sqrt((double)((int64_t)g->nx * g->nx + (int64_t)g->ny * g->ny + (int64_t)g->nz * g->nz));
    long double emitted = 0.0L;
    for (int64_t a = 0; a < n_cat; ++a) {
        T.src_cell[0] = cell[3 * a]; T.src_cell[1] = cell[3 * a + 1]; T.src_cell[2] = cell[3 * a + 2];
        if (!in_box(g, T.src_cell[0], T.src_cell[1], T.src_cell[2])) return ORC_EINVAL;
        T.src_id = (int32_t)a;
        T.L_src = L[a];
        emitted += (long double)L[a];
        for (int64_t pix = 0; pix < 12; ++pix) trace_ray(&T, 0, pix, 0.0, 0.0, L[a] / 12.0);
    }
    if (zero) {
        st->photons_emitted = (double)emitted;
        st->photons_absorbed = (double)T.absorbed;
        st->photons_escaped = (double)T.escaped;
        st->photons_residual = (double)T.residual;
        st->photons_lost = (double)T.lost;
    } else {
        st->photons_emitted += (double)emitted;
        st->photons_absorbed += (double)T.absorbed;
        st->photons_escaped += (double)T.escaped;
        st->photons_residual += (double)T.residual;
        st->photons_lost += (double)T.lost;
    }
    if (log_n_out) *log_n_out = T.log_n;
    return ORC_OK;
}

int orc_trace(const orc_grid *g, const orc_params *p, const void *nH, const void *xHI,
              int64_t n_cat, const int32_t *cell, const double *L, double *gamma, double *heat,
              orc_stats *st, orc_seg *log, int64_t log_cap, int64_t *log_n_out) {
    return trace_catalogue(g, p, nH, xHI, n_cat, cell, L, gamma, heat, st, log, log_cap, log_n_out, 1);
}

/* the same, accumulating into gamma / heat / *st (which the caller zeroes once) */
int orc_trace_add(const orc_grid *g, const orc_params *p, const void *nH, const void *xHI,
                  int64_t n_cat, const int32_t *cell, const double *L, double *gamma, double *heat, orc_stats *st) {
    return trace_catalogue(g, p, nH, xHI, n_cat, cell, L, gamma, heat, st, NULL, 0, NULL, 0);
}

/* the source pass of orc_step alone: dedup + sort, and bubble radii + merge when merging is on */
int orc_catalogue(const orc_grid *g, const orc_params *p, const void *xHI, int64_t n_src, const double *pos,
                  const double *L, orc_stats *st, int32_t *cat_cell, double *cat_L, double *cat_r, int64_t *n_cat);

/* mean ionised fraction over all cells (automerge trigger) */
double orc_mean_ionised(const orc_grid *g, const void *xHI) {
    int64_t ncell = (int64_t)g->nx * g->ny * g->nz;
    long double s = 0.0L;
    for (int64_t i = 0; i < ncell; ++i) s += (long double)(1.0 - fld(xHI, g->field_dtype, i));
    return (double)(s / (long double)ncell);
}

/* The whole step.  cat_* have room for n_src entries; *n_cat receives the catalogue length. */
int orc_catalogue(const orc_grid *g, const orc_params *p, const void *xHI, int64_t n_src, const double *pos,
                  const double *L, orc_stats *st, int32_t *cat_cell, double *cat_L, double *cat_r, int64_t *n_cat) {
    memset(st, 0, sizeof *st);
    int64_t nd = 0;
    int rc = orc_prepare_sources(g, n_src, pos, L, cat_cell, cat_L, &nd);
    if (rc) return rc;
    st->n_src_in = (uint64_t)n_src;
    st->n_src_dedup = (uint64_t)nd;
    for (int64_t a = 0; a < nd; ++a) cat_r[a] = 0.0;
    int do_merge = p->merge == 1 || (p->merge == 2 && orc_mean_ionised(g, xHI) > p->automerge_xmean);
    int64_t nm = nd;
    if (do_merge && nd > 0) {
        int32_t *c2 = malloc((size_t)nd * 3 * sizeof *c2);
        double *L2 = malloc((size_t)nd * sizeof *L2), *r2 = malloc((size_t)nd * sizeof *r2);
        if (!c2 || !L2 || !r2) { free(c2); free(L2); free(r2); return ORC_ENOMEM; }
        rc = orc_bubble_radius(g, p, xHI, nd, cat_cell, cat_r);
        if (!rc) rc = orc_merge(g, p, nd, cat_cell, cat_L, cat_r, c2, L2, r2, &nm);
        if (!rc) {
            memcpy(cat_cell, c2, (size_t)nm * 3 * sizeof *c2);
            memcpy(cat_L, L2, (size_t)nm * sizeof *L2);
            memcpy(cat_r, r2, (size_t)nm * sizeof *r2);
        }
        free(c2); free(L2); free(r2);
        if (rc) return rc;
    }
    st->n_src_merged = (uint64_t)nm;
    *n_cat = nm;
    return ORC_OK;
}

int orc_step(const orc_grid *g, const orc_params *p, const void *nH, const void *xHI,
             int64_t n_src, const double *pos, const double *L,
             double *gamma, double *heat, orc_stats *st,
             int32_t *cat_cell, double *cat_L, double *cat_r, int64_t *n_cat) {
    int rc = orc_catalogue(g, p, xHI, n_src, pos, L, st, cat_cell, cat_L, cat_r, n_cat);
    if (rc) return rc;
    return orc_trace(g, p, nH, xHI, *n_cat, cat_cell, cat_L, gamma, heat, st, NULL, 0, NULL);
}

int orc_sizeof_stats(void) { return (int)sizeof(orc_stats); }
int orc_sizeof_seg(void) { return (int)sizeof(orc_seg); }

/* ------------------------------------------------------------------------------------------ */
/* T1-T3: one RT TIMESTEP = time integration (Sec. 2.3) inside the iterative     */
/* nonlinear solve (Sec. 2.4), "following the approach of [23]" (C2-Ray,        */
/* Mellema et al. 2006): fix x, ray-trace for Gamma (orc_step above); fix Gamma, integrate Eq. 3  */
/* over dt with the semi-analytic, time-averaged solution; iterate until convergence.             */
/* The ray traces inside use the flux that is configured: monochromatic (constant sigma) by       */
/* default, the tau_0 lookup table of PAPER.md:95 after orc_set_spectrum (R32).  Readings R32-R36. */

typedef struct {
    double  dt_s;             /* timestep                                                       */
    double  alpha_cm3_s;      /* recombination coefficient alpha_H(T) of Eq. 3 (isothermal, caller's T) */
    double  coll_cm3_s;       /* collisional ionisation coefficient C_H(T) of Eq. 3              */
    double  clumping;         /* clumping factor C of Eq. 10 (multiplies the recombination rate) */
    double  tol_rel, tol_abs; /* convergence of the time-averaged neutral fraction (R35)         */
    double  unconv_frac;      /* fraction of the cells that may stay unconverged (R35)           */
    int32_t max_iter;         /* outer iterations (RT <-> ODE), >= 1                             */
    int32_t inner_iter;       /* per-cell iterations on the electron density, >= 1 (R34)         */
} orc_ode;

typedef struct {
    int32_t  iterations, converged;
    uint64_t unconverged_cells;    /* in the last iteration                                      */
    uint64_t segments_total;       /* over all iterations                                        */
    double   max_rel_change;       /* of the last iteration: max |dy| / (tol_rel y + tol_abs)    */
} orc_tstats;

/* T2: Eq. 3 in one cell with Gamma fixed, written for the NEUTRAL fraction y = 1 - x:
       dy/dt = -y (Gamma + n_e C_H) + (1 - y) n_e alpha_H C  =  a_rec - y (a_ion + a_rec),
   n_e = <x> n_H held at its time average ([23]'s "time averaging"; the paper's
   "n_e = x n_HI" is read as x n_H, R33).  With constant coefficients the solution is
       y(t) = y_eq + (y0 - y_eq) e^{-t/t_i},  t_i = 1/(a_ion + a_rec),  y_eq = a_rec t_i,
       <y>  = y_eq + (y0 - y_eq) (1 - e^{-dt/t_i}) t_i/dt.
   <y> feeds n_e again, inner_iter times (R34).  yavg_io: in = the current estimate of <y>. */
void orc_ode_cell(const orc_ode *o, double gamma, double nH, double y0, double *yavg_io, double *yend_out) {
    double yavg = *yavg_io, yend = y0;
    for (int it = 0; it < o->inner_iter; ++it) {
        double ne = (1.0 - yavg) * nH;
        double a_ion = gamma + ne * o->coll_cm3_s;
        double a_rec = (ne * o->alpha_cm3_s) * o->clumping;
        double rate = a_ion + a_rec;
        double w = rate * o->dt_s;
        if (!(w > 0.0)) { yend = y0; yavg = y0; break; }           /* nothing acts on the cell */
        double yeq = a_rec / rate;
        double em1 = expm1(-w);                                      /* e^{-w} - 1 */
        yend = yeq + (y0 - yeq) * (1.0 + em1);
        yavg = yeq + (y0 - yeq) * (-em1 / w);
        if (yend < 0.0) yend = 0.0;
        if (yend > 1.0) yend = 1.0;
        if (yavg < 0.0) yavg = 0.0;
        if (yavg > 1.0) yavg = 1.0;
    }
    *yavg_io = yavg;
    *yend_out = yend;
}

/* T3: the iterative solve.  xHI_begin: neutral fraction at the start of the step (fp64).
   xHI_avg: work / output in the FIELD dtype (it is the x_HI field of every ray trace; R36: the
   first trace uses the neutral fraction at the start of the step).  xHI_end: fp64 output.
   gamma / heat: the last iteration's rates.  st: the last iteration's ray statistics. */
int orc_timestep(const orc_grid *g, const orc_params *p, const orc_ode *o, const void *nH,
                 const double *xHI_begin, int64_t n_src, const double *pos, const double *L,
                 double *xHI_end, void *xHI_avg, double *gamma, double *heat, orc_stats *st,
                 orc_tstats *ts, int32_t *cat_cell, double *cat_L, double *cat_r, int64_t *n_cat) {
    if (!(o->dt_s > 0.0) || o->max_iter < 1 || o->inner_iter < 1 || !(o->alpha_cm3_s >= 0.0) ||
        !(o->coll_cm3_s >= 0.0) || !(o->clumping >= 0.0) || !(o->tol_rel >= 0.0) || !(o->tol_abs >= 0.0) || !(o->unconv_frac >= 0.0))
        return ORC_EINVAL;
    const int64_t ncell = (int64_t)g->nx * g->ny * g->nz;
    memset(ts, 0, sizeof *ts);
    for (int64_t c = 0; c < ncell; ++c) {
        if (g->field_dtype) ((float *)xHI_avg)[c] = (float)xHI_begin[c];
        else ((double *)xHI_avg)[c] = xHI_begin[c];
    }
    for (int it = 0; it < o->max_iter; ++it) {
        int rc = orc_step(g, p, nH, xHI_avg, n_src, pos, L, gamma, heat, st, cat_cell, cat_L, cat_r, n_cat);
        if (rc) return rc;
        ts->iterations = it + 1;
        ts->segments_total += st->segments;
        uint64_t bad = 0;
        double worst = 0.0;
        for (int64_t c = 0; c < ncell; ++c) {
            double y_old = fld(xHI_avg, g->field_dtype, c);
            double yavg = y_old, yend;
            orc_ode_cell(o, gamma[c], fld(nH, g->field_dtype, c), xHI_begin[c], &yavg, &yend);
            double y_new;
            if (g->field_dtype) { ((float *)xHI_avg)[c] = (float)yavg; y_new = (double)(float)yavg; }
            else { ((double *)xHI_avg)[c] = yavg; y_new = yavg; }
            xHI_end[c] = yend;
            double lim = o->tol_rel * y_new + o->tol_abs;            /* R35 */
            double dy = fabs(y_new - y_old);
            if (dy > lim) ++bad;
            double q = lim > 0.0 ? dy / lim : (dy > 0.0 ? INFINITY : 0.0);
            if (q > worst) worst = q;
        }
        ts->unconverged_cells = bad;
        ts->max_rel_change = worst;
        if ((double)bad <= o->unconv_frac * (double)ncell) { ts->converged = 1; break; }
    }
    return ORC_OK;
}

int orc_sizeof_ode(void) { return (int)sizeof(orc_ode); }
int orc_sizeof_tstats(void) { return (int)sizeof(orc_tstats); }
