/*
 * mop_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, FP64 CPU oracle for the Onsager-Machlup effective potential
 * V_eff of the metadynamics-of-paths method (arxiv 2501.11962, PAPER.md) and
 * its gradient, written from the paper, sharing no code with the CUDA path.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load this library.
 *
 * What it computes, with the passage each part follows:
 *   O1 pair set        all i<j, not excluded, r_ij < r_c under periodic minimum
 *                      image ("Q atoms ... interacting via U(R)";
 *                      cutoff scheme: "1.2 nm cutoff")
 *   O2 F = -grad U     PAPER.md:40  (F = -nabla_R U); U = LJ 12-6 (+potential
 *                      shift) + reaction-field Coulomb + harmonic bonds/angles
 *                      (the force-field choice is BASELINE.json's north_star)
 *   O3 H s             exact second derivative of U contracted with a direction:
 *                      the eps->0 limit of the bracket in eq. (5)
 *                      [F(R+eps s) - F(R-eps s)]/(4 eps) -> -(1/2) H s
 *   O4 V_eff           eq. (3), K = m nu/(2 dt) and
 *                      L^n = dt/(m nu) F^n  (reading G1 in DESIGN.md: the
 *                      printed L^n is inverted; eqs (5)-(7) require K*L/F = 1/2)
 *   O5 grad V_eff      derivative of eq. (3); equals -(eqs 5,6,7)
 *   O5-FD              the same gradient with the paper's own finite-difference
 *                      Hessian term, eqs (5),(6),(7) as printed (orc_veff_grad_fd)
 *   O6 integrator      velocity Verlet on eq. (4); with the
 *                      Langevin thermostat of the NVT runs (reading G19): orc_step_langevin
 *
 *   O7 MoP bias        S_e2e = s(R^N) - s(R^1) (eq. 8), s = COM distance of
 *                      two atom groups, V(S) a sum of Gaussians
 *
 * Geometry modes (argument `geom`):
 *   0  pure FP64: positions as given, minimum image and r < r_c in double.
 *      Used by the pins (finite differences, invariants, closed forms).
 *   1  "FP32 contract" (reading G8): positions are first rounded to
 *      float; the periodic wrap, the cell index and the in-range predicate
 *      r2 < rc*rc are evaluated in FP32 with a fixed operation order; all the
 *      physics is then done in FP64 on the wrapped float coordinates.  This is
 *      the mode the GPU parity tests compare against, so that neighbour sets
 *      can be compared bit-exactly.
 *
 * Parity pins: every function here is pinned by tests/test_oracle_pins.py
 * (closed forms, finite differences, invariants, brute force); none is
 * "parity unpinned".
 *
 * Build: gcc -O2 -fopenmp -ffp-contract=off -shared -fPIC (see oracle/oracle.py)
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <stdint.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_KE 138.935458 /* kJ mol^-1 nm e^-2 */

typedef struct {
    int n_atoms;
    float box[3];
    float r_cut;
    float eps_rf;   /* <= 0: infinity */
    int lj_shift;
    double dt_path, nu;
    const float *mass, *charge;
    const int *type;
    int n_types;
    const float *c6, *c12;
    int n_bonds;
    const int *bond_ij;
    const float *bond_b0_kb;
    int n_angles;
    const int *angle_ijk;
    const float *angle_t0_kt;
    const int *excl_start, *excl_list;
} orc_system;

/* ------------------------------------------------------------------ */
/* G8: the FP32 expressions (fixed operation order, no contraction).   */
/* ------------------------------------------------------------------ */

/* wrap one coordinate into [0, L):  xw = x - L*floor(x*invL), then fix-ups */
static float orc_wrap1(float x, float L, float invL) {
    float t = x * invL;
    float f = floorf(t);
    float p = L * f;
    float xw = x - p;
    if (xw < 0.0f) xw = xw + L;
    if (xw >= L) xw = xw - L;
    return xw;
}

void orc_wrap(const float *R, int Q, const float box[3], float *xw) {
    for (int d = 0; d < 3; d++) {
        float L = box[d], invL = 1.0f / L;
        for (int i = 0; i < Q; i++) xw[3 * i + d] = orc_wrap1(R[3 * i + d], L, invL);
    }
}

/* Search-grid dimensions (host logic shared by definition):
 * columns in x,y of side ~ (cluster/rho)^(1/3), thin bins of ~bin_z along z.  */
void orc_grid_dims(int Q, const float box[3], int cluster, float bin_z, int dims[3]) {
    double vol = (double)box[0] * (double)box[1] * (double)box[2];
    double side = cbrt((double)cluster * vol / (double)Q);
    for (int d = 0; d < 2; d++) {
        int n = (int)floor((double)box[d] / side);
        if (n < 1) n = 1;
        if (n > 1024) n = 1024;
        dims[d] = n;
    }
    int nz = (int)floor((double)box[2] / (double)bin_z);
    if (nz < 1) nz = 1;
    if (nz > 4096) nz = 4096;
    dims[2] = nz;
}

/* cell id = (cx*ny + cy)*nz + cz, c = min((int)(xw*(n*invL)), n-1) */
void orc_cell_ids(const float *xw, int Q, const float box[3], const int dims[3], int *cell) {
    float sc[3];
    for (int d = 0; d < 3; d++) {
        float invL = 1.0f / box[d];
        sc[d] = (float)dims[d] * invL;
    }
    for (int i = 0; i < Q; i++) {
        int c[3];
        for (int d = 0; d < 3; d++) {
            int v = (int)(xw[3 * i + d] * sc[d]);
            if (v > dims[d] - 1) v = dims[d] - 1;
            c[d] = v;
        }
        cell[i] = (c[0] * dims[1] + c[1]) * dims[2] + c[2];
    }
}

/* stable sort by cell id: perm[k] = original index of the k-th atom (G13) */
void orc_stable_sort_by_cell(const int *cell, int Q, int ncell, int *perm) {
    int *start = (int *)calloc((size_t)ncell + 1, sizeof(int));
    for (int i = 0; i < Q; i++) start[cell[i] + 1]++;
    for (int c = 0; c < ncell; c++) start[c + 1] += start[c];
    for (int i = 0; i < Q; i++) perm[start[cell[i]]++] = i; /* ascending i => stable */
    free(start);
}

/* FP32 pair predicate for a given image shift k (each in {-1,0,1}), reading G8:
 *   d0 = xw_i - xw_j          (one rounding)
 *   d  = d0 - k*L             (k*L exact, one rounding; k = 0: d = d0 exactly)
 *   r2 = fma(dz,dz, fma(dy,dy, dx*dx));   in range iff r2 < rc*rc
 * Both roundings are odd functions of their operands, so swapping the two atoms (k -> -k) gives -d
 * bit for bit and the same r2: membership is a property of the unordered pair, whichever atom an
 * implementation chooses to call i.                                                              */
static int orc_pred_f32(const float *xi, const float *xj, const float box[3], const int k[3],
                        float rc2, float *r2out) {
    float d[3];
    for (int a = 0; a < 3; a++) {
        float s = (float)k[a] * box[a];
        float d0 = xi[a] - xj[a];
        d[a] = d0 - s;
    }
    float r2 = fmaf(d[2], d[2], fmaf(d[1], d[1], d[0] * d[0]));
    if (r2out) *r2out = r2;
    return r2 < rc2;
}

/* nearest image index per dimension, FP32: k = rintf((xi-xj)*invL) */
static void orc_image_f32(const float *xi, const float *xj, const float box[3], int k[3]) {
    for (int a = 0; a < 3; a++) {
        float invL = 1.0f / box[a];
        float d0 = xi[a] - xj[a];
        k[a] = (int)rintf(d0 * invL);
    }
}

/* ------------------------------------------------------------------ */
/* exclusions                                                           */
/* ------------------------------------------------------------------ */
static int orc_excluded(const orc_system *s, int i, int j) {
    if (!s->excl_start) return 0;
    for (int e = s->excl_start[i]; e < s->excl_start[i + 1]; e++)
        if (s->excl_list[e] == j) return 1;
    return 0;
}

/* ------------------------------------------------------------------ */
/* O1: pair enumeration.  The callback receives i<j, the separation     */
/* d = r_i - r_j (minimum image, double) and r2 = d.d (double).         */
/* ------------------------------------------------------------------ */
typedef void (*orc_pair_fn)(void *ctx, int i, int j, const double d[3], double r2);

typedef struct {
    const orc_system *s;
    int geom;
    const double *x;  /* geom 0: positions as given; geom 1: wrapped floats promoted */
    const float *xw;  /* geom 1 only */
    double boxd[3];
    double rc2d;
    float rc2f;
} orc_geom;

/* test one candidate pair; returns 1 and fills d,r2 when in range and not excluded */
static int orc_pair_test(const orc_geom *g, int i, int j, double d[3], double *r2) {
    if (g->geom == 0) {
        double rr = 0.0;
        for (int a = 0; a < 3; a++) {
            double dd = g->x[3 * i + a] - g->x[3 * j + a];
            dd -= g->boxd[a] * rint(dd / g->boxd[a]);
            d[a] = dd;
            rr += dd * dd;
        }
        *r2 = rr;
        return rr < g->rc2d;
    } else {
        int k[3];
        orc_image_f32(g->xw + 3 * i, g->xw + 3 * j, g->s->box, k);
        if (!orc_pred_f32(g->xw + 3 * i, g->xw + 3 * j, g->s->box, k, g->rc2f, NULL)) return 0;
        double rr = 0.0;
        for (int a = 0; a < 3; a++) {
            double dd = ((double)g->xw[3 * i + a] - (double)g->xw[3 * j + a]) - (double)k[a] * g->boxd[a];
            d[a] = dd;
            rr += dd * dd;
        }
        *r2 = rr;
        return 1;
    }
}

/* brute force: every i<j; in geom 1 every one of the 27 images is tried with the
 * FP32 predicate (at most one can be in range when min(box) >= 2 r_c).           */
static void orc_pairs_brute(const orc_geom *g, orc_pair_fn fn, void *ctx) {
    const orc_system *s = g->s;
    int Q = s->n_atoms;
    for (int i = 0; i < Q; i++)
        for (int j = i + 1; j < Q; j++) {
            if (orc_excluded(s, i, j)) continue;
            double d[3], r2;
            if (g->geom == 0) {
                if (orc_pair_test(g, i, j, d, &r2)) fn(ctx, i, j, d, r2);
            } else {
                int k[3];
                for (k[0] = -1; k[0] <= 1; k[0]++)
                    for (k[1] = -1; k[1] <= 1; k[1]++)
                        for (k[2] = -1; k[2] <= 1; k[2]++) {
                            if (!orc_pred_f32(g->xw + 3 * i, g->xw + 3 * j, s->box, k, g->rc2f, NULL)) continue;
                            r2 = 0.0;
                            for (int a = 0; a < 3; a++) {
                                d[a] = ((double)g->xw[3 * i + a] - (double)g->xw[3 * j + a]) - (double)k[a] * g->boxd[a];
                                r2 += d[a] * d[a];
                            }
                            fn(ctx, i, j, d, r2);
                        }
            }
        }
}

/* the oracle's own linked-cell list: cells of side >= r_c, 27-cell stencil with
 * duplicate cells removed when a dimension has fewer than 3 cells.               */
static void orc_pairs_cell(const orc_geom *g, orc_pair_fn fn, void *ctx) {
    const orc_system *s = g->s;
    int Q = s->n_atoms;
    int nc[3];
    for (int a = 0; a < 3; a++) {
        nc[a] = (int)floor(g->boxd[a] / (double)s->r_cut);
        if (nc[a] < 1) nc[a] = 1;
    }
    int ncell = nc[0] * nc[1] * nc[2];
    int *head = (int *)malloc(sizeof(int) * (size_t)ncell);
    int *next = (int *)malloc(sizeof(int) * (size_t)Q);
    int *cidx = (int *)malloc(sizeof(int) * (size_t)Q * 3);
    for (int c = 0; c < ncell; c++) head[c] = -1;
    /* insert in descending i so that each chain is ascending in i */
    for (int i = Q - 1; i >= 0; i--) {
        int c[3];
        for (int a = 0; a < 3; a++) {
            double x = g->x[3 * i + a];
            double f = x / g->boxd[a];
            f -= floor(f);
            int v = (int)(f * nc[a]);
            if (v >= nc[a]) v = nc[a] - 1;
            if (v < 0) v = 0;
            c[a] = v;
            cidx[3 * i + a] = v;
        }
        int ci = (c[0] * nc[1] + c[1]) * nc[2] + c[2];
        next[i] = head[ci];
        head[ci] = i;
    }
    for (int i = 0; i < Q; i++) {
        int seen[27], nseen = 0;
        for (int ox = -1; ox <= 1; ox++)
            for (int oy = -1; oy <= 1; oy++)
                for (int oz = -1; oz <= 1; oz++) {
                    int c0 = ((cidx[3 * i + 0] + ox) % nc[0] + nc[0]) % nc[0];
                    int c1 = ((cidx[3 * i + 1] + oy) % nc[1] + nc[1]) % nc[1];
                    int c2 = ((cidx[3 * i + 2] + oz) % nc[2] + nc[2]) % nc[2];
                    int cj = (c0 * nc[1] + c1) * nc[2] + c2;
                    int dup = 0;
                    for (int q = 0; q < nseen; q++)
                        if (seen[q] == cj) dup = 1;
                    if (dup) continue;
                    seen[nseen++] = cj;
                    for (int j = head[cj]; j >= 0; j = next[j]) {
                        if (j <= i) continue;
                        if (orc_excluded(s, i, j)) continue;
                        double d[3], r2;
                        if (orc_pair_test(g, i, j, d, &r2)) fn(ctx, i, j, d, r2);
                    }
                }
    }
    free(head);
    free(next);
    free(cidx);
}

/* prepare geometry for one bead.  R: [Q][3] doubles as given by the caller.
 * geom 1: round to float, wrap in FP32; x = wrapped floats promoted.             */
static void orc_geom_init(orc_geom *g, const orc_system *s, int geom, const double *R, double *xbuf,
                          float *xwbuf) {
    g->s = s;
    g->geom = geom;
    for (int a = 0; a < 3; a++) g->boxd[a] = (double)s->box[a];
    g->rc2d = (double)s->r_cut * (double)s->r_cut;
    g->rc2f = s->r_cut * s->r_cut;
    int Q = s->n_atoms;
    if (geom == 0) {
        g->x = R;
        g->xw = NULL;
    } else {
        float *Rf = (float *)malloc(sizeof(float) * 3 * (size_t)Q);
        for (int i = 0; i < 3 * Q; i++) Rf[i] = (float)R[i];
        orc_wrap(Rf, Q, s->box, xwbuf);
        free(Rf);
        for (int i = 0; i < 3 * Q; i++) xbuf[i] = (double)xwbuf[i];
        g->x = xbuf;
        g->xw = xwbuf;
    }
}

static void orc_for_pairs(const orc_geom *g, int brute, orc_pair_fn fn, void *ctx) {
    if (brute)
        orc_pairs_brute(g, fn, ctx);
    else
        orc_pairs_cell(g, fn, ctx);
}

/* exported: list the in-range pairs of one bead; returns the count, writes up to
 * cap pairs (i<j, original indices) into pairs[2*k], pairs[2*k+1].               */
typedef struct {
    int *pairs;
    long cap, n;
} orc_collect;
static void orc_collect_fn(void *ctx, int i, int j, const double d[3], double r2) {
    (void)d;
    (void)r2;
    orc_collect *c = (orc_collect *)ctx;
    if (c->n < c->cap) {
        c->pairs[2 * c->n] = i;
        c->pairs[2 * c->n + 1] = j;
    }
    c->n++;
}
long orc_pairs(const orc_system *s, const double *R, int geom, int brute, int *pairs, long cap) {
    int Q = s->n_atoms;
    double *xb = (double *)malloc(sizeof(double) * 3 * (size_t)Q);
    float *xw = (float *)malloc(sizeof(float) * 3 * (size_t)Q);
    orc_geom g;
    orc_geom_init(&g, s, geom, R, xb, xw);
    orc_collect c = {pairs, cap, 0};
    orc_for_pairs(&g, brute, orc_collect_fn, &c);
    free(xb);
    free(xw);
    return c.n;
}

/* ------------------------------------------------------------------ */
/* O2 / O3: pair potentials                                             */
/* ------------------------------------------------------------------ */
typedef struct {
    const orc_system *s;
    double krf, crf;
    double *F;        /* [Q][3] or NULL */
    double u_lj, u_coul;
    const double *sv; /* direction s [Q][3] (HVP) or NULL */
    double *Hs;       /* [Q][3] or NULL */
    long npairs;
} orc_nb;

static void orc_rf_consts(const orc_system *s, double *krf, double *crf) {
    double rc = (double)s->r_cut;
    if (s->eps_rf > 0.0f) {
        double e = (double)s->eps_rf;
        *krf = (e - 1.0) / ((2.0 * e + 1.0) * rc * rc * rc);
    } else {
        *krf = 1.0 / (2.0 * rc * rc * rc);
    }
    *crf = 1.0 / rc + (*krf) * rc * rc;
}

/* u(r), g = u'/r, h = (u'' - u'/r)/r^2 for LJ + reaction field */
static void orc_nb_scalars(const orc_nb *nb, int i, int j, double r2, double *u_lj, double *u_c, double *g,
                           double *h) {
    const orc_system *s = nb->s;
    int ti = s->type[i], tj = s->type[j];
    double c6 = (double)s->c6[ti * s->n_types + tj];
    double c12 = (double)s->c12[ti * s->n_types + tj];
    double qq = ORC_KE * (double)s->charge[i] * (double)s->charge[j];
    double r = sqrt(r2);
    double ir2 = 1.0 / r2;
    double ir6 = ir2 * ir2 * ir2;
    double ir12 = ir6 * ir6;
    double ulj = c12 * ir12 - c6 * ir6;
    if (s->lj_shift) {
        double rc = (double)s->r_cut;
        double irc6 = 1.0 / (rc * rc * rc * rc * rc * rc);
        ulj -= c12 * irc6 * irc6 - c6 * irc6;
    }
    *u_lj = ulj;
    *u_c = qq * (1.0 / r + nb->krf * r2 - nb->crf);
    /* u'/r */
    double g_lj = (-12.0 * c12 * ir12 + 6.0 * c6 * ir6) * ir2;
    double g_c = qq * (-1.0 / (r2 * r) + 2.0 * nb->krf);
    *g = g_lj + g_c;
    /* (u'' - u'/r)/r^2 */
    double h_lj = (168.0 * c12 * ir12 - 48.0 * c6 * ir6) * ir2 * ir2;
    double h_c = 3.0 * qq / (r2 * r2 * r);
    *h = h_lj + h_c;
}

static void orc_nb_fn(void *ctx, int i, int j, const double d[3], double r2) {
    orc_nb *nb = (orc_nb *)ctx;
    double ulj, uc, g, h;
    orc_nb_scalars(nb, i, j, r2, &ulj, &uc, &g, &h);
    nb->npairs++;
    nb->u_lj += ulj;
    nb->u_coul += uc;
    if (nb->F) {
        /* F_i = -u'(r) d/r = -g d */
        for (int a = 0; a < 3; a++) {
            nb->F[3 * i + a] -= g * d[a];
            nb->F[3 * j + a] += g * d[a];
        }
    }
    if (nb->Hs) {
        double del[3], dd = 0.0;
        for (int a = 0; a < 3; a++) {
            del[a] = nb->sv[3 * i + a] - nb->sv[3 * j + a];
            dd += d[a] * del[a];
        }
        for (int a = 0; a < 3; a++) {
            double t = h * dd * d[a] + g * del[a];
            nb->Hs[3 * i + a] += t;
            nb->Hs[3 * j + a] -= t;
        }
    }
}

/* bonded terms use the caller's (unwrapped) coordinates with a minimum image */
static void orc_mi(const double *xi, const double *xj, const double box[3], double d[3]) {
    for (int a = 0; a < 3; a++) {
        double dd = xi[a] - xj[a];
        dd -= box[a] * rint(dd / box[a]);
        d[a] = dd;
    }
}

static void orc_bonded(const orc_system *s, const double *x, const double box[3], double *F, const double *sv,
                       double *Hs, double *u_bond, double *u_angle) {
    double ub = 0.0, ua = 0.0;
    for (int b = 0; b < s->n_bonds; b++) {
        int i = s->bond_ij[2 * b], j = s->bond_ij[2 * b + 1];
        double b0 = (double)s->bond_b0_kb[2 * b], kb = (double)s->bond_b0_kb[2 * b + 1];
        double d[3];
        orc_mi(x + 3 * i, x + 3 * j, box, d);
        double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
        ub += 0.5 * kb * (r - b0) * (r - b0);
        double g = kb * (1.0 - b0 / r); /* u'/r */
        double h = kb * b0 / (r * r * r); /* (u''-u'/r)/r^2 */
        if (F)
            for (int a = 0; a < 3; a++) {
                F[3 * i + a] -= g * d[a];
                F[3 * j + a] += g * d[a];
            }
        if (Hs) {
            double del[3], dd = 0.0;
            for (int a = 0; a < 3; a++) {
                del[a] = sv[3 * i + a] - sv[3 * j + a];
                dd += d[a] * del[a];
            }
            for (int a = 0; a < 3; a++) {
                double t = h * dd * d[a] + g * del[a];
                Hs[3 * i + a] += t;
                Hs[3 * j + a] -= t;
            }
        }
    }
    for (int t = 0; t < s->n_angles; t++) {
        int i = s->angle_ijk[3 * t], j = s->angle_ijk[3 * t + 1], k = s->angle_ijk[3 * t + 2];
        double t0 = (double)s->angle_t0_kt[2 * t], kt = (double)s->angle_t0_kt[2 * t + 1];
        double a[3], b[3];
        orc_mi(x + 3 * i, x + 3 * j, box, a);
        orc_mi(x + 3 * k, x + 3 * j, box, b);
        double la = sqrt(a[0] * a[0] + a[1] * a[1] + a[2] * a[2]);
        double lb = sqrt(b[0] * b[0] + b[1] * b[1] + b[2] * b[2]);
        double ah[3], bh[3];
        for (int q = 0; q < 3; q++) {
            ah[q] = a[q] / la;
            bh[q] = b[q] / lb;
        }
        double c = ah[0] * bh[0] + ah[1] * bh[1] + ah[2] * bh[2];
        if (c > 1.0) c = 1.0;
        if (c < -1.0) c = -1.0;
        double th = acos(c);
        double sg = sqrt(1.0 - c * c);
        ua += 0.5 * kt * (th - t0) * (th - t0);
        double p[3], qv[3], ga[3], gb[3];
        for (int q = 0; q < 3; q++) {
            p[q] = bh[q] - c * ah[q];
            qv[q] = ah[q] - c * bh[q];
            ga[q] = -p[q] / (la * sg); /* d theta / d a */
            gb[q] = -qv[q] / (lb * sg); /* d theta / d b */
        }
        double pref = kt * (th - t0);
        if (F)
            for (int q = 0; q < 3; q++) {
                double fi = -pref * ga[q], fk = -pref * gb[q];
                F[3 * i + q] += fi;
                F[3 * k + q] += fk;
                F[3 * j + q] -= fi + fk;
            }
        if (Hs) {
            double da[3], db[3];
            for (int q = 0; q < 3; q++) {
                da[q] = sv[3 * i + q] - sv[3 * j + q];
                db[q] = sv[3 * k + q] - sv[3 * j + q];
            }
            double dth = 0.0, dla = 0.0, dlb = 0.0;
            for (int q = 0; q < 3; q++) {
                dth += ga[q] * da[q] + gb[q] * db[q];
                dla += ah[q] * da[q];
                dlb += bh[q] * db[q];
            }
            double dah[3], dbh[3];
            for (int q = 0; q < 3; q++) {
                dah[q] = (da[q] - ah[q] * dla) / la;
                dbh[q] = (db[q] - bh[q] * dlb) / lb;
            }
            double dc = 0.0;
            for (int q = 0; q < 3; q++) dc += dah[q] * bh[q] + ah[q] * dbh[q];
            double dsg = -c * dc / sg;
            for (int q = 0; q < 3; q++) {
                double dp = dbh[q] - dc * ah[q] - c * dah[q];
                double dq = dah[q] - dc * bh[q] - c * dbh[q];
                double dga = -dp / (la * sg) + p[q] * (dla * sg + la * dsg) / ((la * sg) * (la * sg));
                double dgb = -dq / (lb * sg) + qv[q] * (dlb * sg + lb * dsg) / ((lb * sg) * (lb * sg));
                double hi = kt * dth * ga[q] + pref * dga;
                double hk = kt * dth * gb[q] + pref * dgb;
                Hs[3 * i + q] += hi;
                Hs[3 * k + q] += hk;
                Hs[3 * j + q] -= hi + hk;
            }
        }
    }
    if (u_bond) *u_bond = ub;
    if (u_angle) *u_angle = ua;
}

/* exported: physical force, energy terms and (optionally) H s for ONE bead.
 * R [Q][3] doubles; F, Hs [Q][3] doubles (may be NULL); sv [Q][3] or NULL.
 * u_out[4] = {U_lj, U_coul, U_bond, U_angle}; returns in-range pair count.       */
long orc_bead(const orc_system *s, const double *R, int geom, int brute, double *F, const double *sv,
              double *Hs, double *u_out) {
    int Q = s->n_atoms;
    double *xb = (double *)malloc(sizeof(double) * 3 * (size_t)Q);
    float *xw = (float *)malloc(sizeof(float) * 3 * (size_t)Q);
    double *xu = (double *)malloc(sizeof(double) * 3 * (size_t)Q);
    orc_geom g;
    orc_geom_init(&g, s, geom, R, xb, xw);
    /* bonded terms: caller coordinates (rounded to float in geom 1), not wrapped */
    for (int i = 0; i < 3 * Q; i++) xu[i] = geom ? (double)(float)R[i] : R[i];
    if (F) memset(F, 0, sizeof(double) * 3 * (size_t)Q);
    if (Hs) memset(Hs, 0, sizeof(double) * 3 * (size_t)Q);
    orc_nb nb;
    memset(&nb, 0, sizeof nb);
    nb.s = s;
    orc_rf_consts(s, &nb.krf, &nb.crf);
    nb.F = F;
    nb.sv = sv;
    nb.Hs = (sv ? Hs : NULL);
    orc_for_pairs(&g, brute, orc_nb_fn, &nb);
    double ub = 0.0, ua = 0.0;
    orc_bonded(s, xu, g.boxd, F, sv, (sv ? Hs : NULL), &ub, &ua);
    if (u_out) {
        u_out[0] = nb.u_lj;
        u_out[1] = nb.u_coul;
        u_out[2] = ub;
        u_out[3] = ua;
    }
    free(xb);
    free(xw);
    free(xu);
    return nb.npairs;
}

/* ------------------------------------------------------------------ */
/* O4 + O5: V_eff (eq. 3) and its gradient                              */
/* ------------------------------------------------------------------ */
/* R [N][Q][3] doubles.  Outputs (any may be NULL):
 *   grad [N][Q][3]  dV_eff/dR^n  (= -F_eff^n of eqs 5,6,7)
 *   Fout, eta, Heta [max(N-1,1)][Q][3]
 *   parts[4] = {U(R^1), E_spring, total in-range pairs over force beads, 0}
 * returns V_eff.                                                                  */
double orc_veff_grad(const orc_system *s, int N, const double *R, int geom, int brute, double *grad,
                     double *Fout, double *eta_out, double *Heta_out, double *parts) {
    int Q = s->n_atoms;
    size_t bead = 3 * (size_t)Q;
    int nf = (N > 1) ? N - 1 : 1; /* beads that need F (G6: bead N does not) */
    double *F = (double *)malloc(sizeof(double) * bead * (size_t)nf);
    double *eta = (double *)calloc(bead * (size_t)nf, sizeof(double));
    double *Heta = (double *)calloc(bead * (size_t)nf, sizeof(double));
    double *U = (double *)calloc((size_t)nf * 4, sizeof(double));
    long *np = (long *)calloc((size_t)nf, sizeof(long));
    /* positions entering the spring term: caller coordinates, rounded to float in geom 1 */
    double *X = (double *)malloc(sizeof(double) * bead * (size_t)N);
    for (size_t i = 0; i < bead * (size_t)N; i++) X[i] = geom ? (double)(float)R[i] : R[i];

#pragma omp parallel for schedule(dynamic, 1)
    for (int n = 0; n < nf; n++) np[n] = orc_bead(s, R + bead * n, geom, brute, F + bead * n, NULL, NULL, U + 4 * n);

    double e_spring = 0.0;
    if (N > 1) {
        for (int n = 0; n < N - 1; n++)
            for (int i = 0; i < Q; i++) {
                double m = (double)s->mass[i];
                double a = s->dt_path / (m * s->nu);      /* L^n_i = a_i F^n_i   (G1) */
                double K = m * s->nu / (2.0 * s->dt_path);
                for (int q = 0; q < 3; q++) {
                    size_t o = bead * n + 3 * (size_t)i + q;
                    double e = (X[o + bead] - X[o]) - a * F[o];
                    eta[o] = e;
                    e_spring += 0.5 * K * e * e;
                }
            }
#pragma omp parallel for schedule(dynamic, 1)
        for (int n = 0; n < N - 1; n++)
            orc_bead(s, R + bead * n, geom, brute, NULL, eta + bead * n, Heta + bead * n, NULL);
    }
    double U1 = U[0] + U[1] + U[2] + U[3];
    double veff = U1 + e_spring;
    if (grad) {
        for (int n = 0; n < N; n++)
            for (int i = 0; i < Q; i++) {
                double m = (double)s->mass[i];
                double K = m * s->nu / (2.0 * s->dt_path);
                for (int q = 0; q < 3; q++) {
                    size_t o = bead * n + 3 * (size_t)i + q;
                    double gsum = 0.0;
                    if (n == 0) gsum -= F[o];                              /* dU(R^1)/dR^1        */
                    if (n > 0) gsum += K * eta[o - bead];                  /* spring n-1 -> n     */
                    if (n < N - 1) gsum += -K * eta[o] + 0.5 * Heta[o];    /* K a_i = 1/2 exactly */
                    grad[o] = gsum;
                }
            }
    }
    long tot = 0;
    for (int n = 0; n < nf; n++) tot += np[n];
    if (parts) {
        parts[0] = U1;
        parts[1] = e_spring;
        parts[2] = (double)tot;
        parts[3] = 0.0;
    }
    if (Fout) memcpy(Fout, F, sizeof(double) * bead * (size_t)nf);
    if (eta_out) memcpy(eta_out, eta, sizeof(double) * bead * (size_t)nf);
    if (Heta_out) memcpy(Heta_out, Heta, sizeof(double) * bead * (size_t)nf);
    free(F);
    free(eta);
    free(Heta);
    free(U);
    free(np);
    free(X);
    return veff;
}

/* ------------------------------------------------------------------ */
/* O5-FD: the paper's effective force as printed, eqs (5),(6),(7)      */
/* (PAPER.md:61-70), with the Hessian term as the finite difference     */
/*   [F(R^n + eps eta^n) - F(R^n - eps eta^n)] / (4 eps),               */
/*   eta^n = R^{n+1} - R^n - L^n  (L^n = a F^n, reading G1) */
/* eps is the paper's dimensionless epsilon, the same for every bead.   */
/* grad [N][Q][3] receives -F_eff^n; returns V_eff (eq. 3).             */
/* In geom 1 the displaced coordinates are rounded to float like every  */
/* other position (inside orc_bead) before wrap, predicate and physics. */
/* ------------------------------------------------------------------ */
double orc_veff_grad_fd(const orc_system *s, int N, const double *R, double eps, int geom, int brute, double *grad) {
    int Q = s->n_atoms;
    size_t bead = 3 * (size_t)Q;
    int nf = (N > 1) ? N - 1 : 1;
    double *F = (double *)malloc(sizeof(double) * bead * (size_t)nf);
    double *Fp = (double *)calloc(bead * (size_t)nf, sizeof(double));
    double *Fm = (double *)calloc(bead * (size_t)nf, sizeof(double));
    double *Rp = (double *)malloc(sizeof(double) * bead * (size_t)nf);
    double *Rm = (double *)malloc(sizeof(double) * bead * (size_t)nf);
    double *U = (double *)calloc((size_t)nf * 4, sizeof(double));
    double *X = (double *)malloc(sizeof(double) * bead * (size_t)N);
    for (size_t i = 0; i < bead * (size_t)N; i++) X[i] = geom ? (double)(float)R[i] : R[i];
#pragma omp parallel for schedule(dynamic, 1)
    for (int n = 0; n < nf; n++) orc_bead(s, R + bead * n, geom, brute, F + bead * n, NULL, NULL, U + 4 * n);
    double e_spring = 0.0;
    if (N > 1) {
        for (int n = 0; n < N - 1; n++)
            for (int i = 0; i < Q; i++) {
                double m = (double)s->mass[i];
                double a = s->dt_path / (m * s->nu);
                double K = m * s->nu / (2.0 * s->dt_path);
                for (int q = 0; q < 3; q++) {
                    size_t o = bead * n + 3 * (size_t)i + q;
                    double e = (X[o + bead] - X[o]) - a * F[o]; /* eta^n */
                    e_spring += 0.5 * K * e * e;
                    Rp[o] = X[o] + eps * e;                     /* paper kernel 2 */
                    Rm[o] = X[o] - eps * e;
                }
            }
#pragma omp parallel for schedule(dynamic, 1)
        for (int n = 0; n < 2 * (N - 1); n++) {
            int b = n >> 1;
            if (n & 1) orc_bead(s, Rm + bead * b, geom, brute, Fm + bead * b, NULL, NULL, NULL);
            else orc_bead(s, Rp + bead * b, geom, brute, Fp + bead * b, NULL, NULL, NULL);
        }
    }
    double veff = U[0] + U[1] + U[2] + U[3] + e_spring;
    if (grad) {
        for (int n = 0; n < N; n++)
            for (int i = 0; i < Q; i++) {
                double m = (double)s->mass[i];
                double K = m * s->nu / (2.0 * s->dt_path);
                for (int q = 0; q < 3; q++) {
                    size_t o = bead * n + 3 * (size_t)i + q;
                    double feff;
                    if (N == 1) {
                        feff = F[o];                                                   /* V_eff = U(R^1) */
                    } else if (n == 0) {                                               /* eq. (6) */
                        feff = 0.5 * F[o] + K * (X[o + bead] - X[o]) + (Fp[o] - Fm[o]) / (4.0 * eps);
                    } else if (n < N - 1) {                                            /* eq. (5) */
                        feff = -K * (2.0 * X[o] - X[o - bead] - X[o + bead]) + 0.5 * (F[o - bead] - F[o]) +
                               (Fp[o] - Fm[o]) / (4.0 * eps);
                    } else {                                                           /* eq. (7) */
                        feff = -K * (X[o] - X[o - bead]) + 0.5 * F[o - bead];
                    }
                    grad[o] = -feff;
                }
            }
    }
    free(F), free(Fp), free(Fm), free(Rp), free(Rm), free(U), free(X);
    return veff;
}

/* ------------------------------------------------------------------ */
/* O6: velocity Verlet on eq. (4), fictitious mass = physical mass (G4) */
/* ------------------------------------------------------------------ */
/* R, V [N][Q][3] doubles updated in place.  energies[3*(n_steps+1)] (may be NULL)
 * receives {V_eff, E_kin, total} before the first step and after every step.      */
void orc_step(const orc_system *s, int N, double *R, double *V, double dt, int n_steps, int geom, int brute,
              double *energies) {
    int Q = s->n_atoms;
    size_t tot = 3 * (size_t)Q * (size_t)N;
    double *G = (double *)malloc(sizeof(double) * tot);
    double veff = orc_veff_grad(s, N, R, geom, brute, G, NULL, NULL, NULL, NULL);
    for (int st = 0; st <= n_steps; st++) {
        if (energies) {
            double ek = 0.0;
            for (size_t o = 0; o < tot; o++) {
                double m = (double)s->mass[(o / 3) % (size_t)Q];
                ek += 0.5 * m * V[o] * V[o];
            }
            energies[3 * st] = veff;
            energies[3 * st + 1] = ek;
            energies[3 * st + 2] = veff + ek;
        }
        if (st == n_steps) break;
        for (size_t o = 0; o < tot; o++) {
            double m = (double)s->mass[(o / 3) % (size_t)Q];
            V[o] += 0.5 * dt * (-G[o]) / m;
            R[o] += dt * V[o];
        }
        veff = orc_veff_grad(s, N, R, geom, brute, G, NULL, NULL, NULL, NULL);
        for (size_t o = 0; o < tot; o++) {
            double m = (double)s->mass[(o / 3) % (size_t)Q];
            V[o] += 0.5 * dt * (-G[o]) / m;
        }
    }
    free(G);
}

/* ------------------------------------------------------------------ */
/* O6-NVT: path MD with a Langevin thermostat ("the Langevin */
/* thermostat, as implemented in GROMACS, damping coefficient 0.25 fs^-1", */
/* Fig. 4b).  The paper gives no discretisation; reading G19 */
/* (DESIGN.md): one velocity-Verlet step of eq. (4), then the exact        */
/* Ornstein-Uhlenbeck velocity update over dt                              */
/*    v <- c v + sqrt((1 - c^2) kT / m) xi,   c = exp(-gamma dt),          */
/* xi ~ N(0,1) from a counter-based generator keyed by (seed, step, index  */
/* of the coordinate in [N][Q][3]): 64-bit mix -> two 32-bit uniforms ->   */
/* Box-Muller.  gamma = 0 reproduces orc_step exactly.                     */
/* ------------------------------------------------------------------ */
static uint64_t orc_mix64(uint64_t z) { /* SplitMix64 finaliser (Steele, Lea, Flood 2014) */
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}
/* the 64 random bits of (seed, step, idx) */
uint64_t orc_noise_bits(uint64_t seed, uint64_t step, uint64_t idx) {
    return orc_mix64(orc_mix64(seed + 0x9E3779B97F4A7C15ULL * (step + 1)) ^ (idx * 0xD1342543DE82EF95ULL + 1));
}
double orc_noise_normal(uint64_t seed, uint64_t step, uint64_t idx) {
    uint64_t b = orc_noise_bits(seed, step, idx);
    double u1 = ((double)(uint32_t)(b >> 32) + 0.5) / 4294967296.0; /* in (0,1) */
    double u2 = ((double)(uint32_t)b + 0.5) / 4294967296.0;
    return sqrt(-2.0 * log(u1)) * cos(6.283185307179586476925 * u2);
}
/* energies[3*(n_steps+1)] as in orc_step (kinetic energy after the thermostat update) */
void orc_step_langevin(const orc_system *s, int N, double *R, double *V, double dt, int n_steps, double gamma,
                       double kT, uint64_t seed, uint64_t step0, int geom, int brute, double *energies) {
    int Q = s->n_atoms;
    size_t tot = 3 * (size_t)Q * (size_t)N;
    double *G = (double *)malloc(sizeof(double) * tot);
    double veff = orc_veff_grad(s, N, R, geom, brute, G, NULL, NULL, NULL, NULL);
    double c = exp(-gamma * dt), amp = sqrt(1.0 - c * c);
    for (int st = 0; st <= n_steps; st++) {
        if (energies) {
            double ek = 0.0;
            for (size_t o = 0; o < tot; o++) ek += 0.5 * (double)s->mass[(o / 3) % (size_t)Q] * V[o] * V[o];
            energies[3 * st] = veff, energies[3 * st + 1] = ek, energies[3 * st + 2] = veff + ek;
        }
        if (st == n_steps) break;
        for (size_t o = 0; o < tot; o++) {
            double m = (double)s->mass[(o / 3) % (size_t)Q];
            V[o] += 0.5 * dt * (-G[o]) / m;
            R[o] += dt * V[o];
        }
        veff = orc_veff_grad(s, N, R, geom, brute, G, NULL, NULL, NULL, NULL);
        for (size_t o = 0; o < tot; o++) {
            double m = (double)s->mass[(o / 3) % (size_t)Q];
            V[o] += 0.5 * dt * (-G[o]) / m;
            if (gamma > 0.0) V[o] = c * V[o] + amp * sqrt(kT / m) * orc_noise_normal(seed, step0 + (uint64_t)st, (uint64_t)o);
        }
    }
    free(G);
}

/* ------------------------------------------------------------------ */
/* O7: the metadynamics-of-paths bias.            */
/*   CV   S_e2e = s(R^N) - s(R^1)                      eq. (8)          */
/*   s(R) = distance between the centres of mass of two atom groups     */
/*          ("the distance between the center of mass of the ligand and */
/*          the binding pocket"), minimum image of the    */
/*          COM difference; every group is whole in the given coords    */
/*   V(S) = sum_k w exp(-(S - S_k)^2 / (2 sigma^2))   (PAPER.md:80-82:  */
/*          "a sum of Gaussian functions deposited along the CV")       */
/* ------------------------------------------------------------------ */
/* s(X) for one bead X [Q][3]; dsdr [Q][3] (may be NULL) receives ds/dr_i (zero off the groups) */
double orc_cv_com_distance(const orc_system *s, const double *X, const int *ga, int na, const int *gb, int nb,
                           double *dsdr) {
    double ca[3] = {0, 0, 0}, cb[3] = {0, 0, 0}, ma = 0.0, mb = 0.0, d[3];
    for (int k = 0; k < na; k++) {
        double m = (double)s->mass[ga[k]];
        ma += m;
        for (int q = 0; q < 3; q++) ca[q] += m * X[3 * (size_t)ga[k] + q];
    }
    for (int k = 0; k < nb; k++) {
        double m = (double)s->mass[gb[k]];
        mb += m;
        for (int q = 0; q < 3; q++) cb[q] += m * X[3 * (size_t)gb[k] + q];
    }
    double r2 = 0.0;
    for (int q = 0; q < 3; q++) {
        double L = (double)s->box[q];
        d[q] = ca[q] / ma - cb[q] / mb;
        d[q] -= L * floor(d[q] / L + 0.5);
        r2 += d[q] * d[q];
    }
    double r = sqrt(r2);
    if (dsdr) {
        memset(dsdr, 0, sizeof(double) * 3 * (size_t)s->n_atoms);
        if (r > 0.0) {
            for (int k = 0; k < na; k++)
                for (int q = 0; q < 3; q++) dsdr[3 * (size_t)ga[k] + q] += (double)s->mass[ga[k]] / ma * d[q] / r;
            for (int k = 0; k < nb; k++)
                for (int q = 0; q < 3; q++) dsdr[3 * (size_t)gb[k] + q] -= (double)s->mass[gb[k]] / mb * d[q] / r;
        }
    }
    return r;
}
/* V(S_e2e) of a path R [N][Q][3] (N >= 2); grad_add [N][Q][3] (may be NULL) receives dV/dR^n (zero on the interior
 * beads: the CV touches beads 1 and N only); out[3] = {S_e2e, s(R^1), s(R^N)} (may be NULL).  Returns V.            */
double orc_bias(const orc_system *s, int N, const double *R, const int *ga, int na, const int *gb, int nb,
                const double *hills, int nh, double sigma, double w, double *grad_add, double *out) {
    size_t bead = 3 * (size_t)s->n_atoms;
    double *d1 = (double *)malloc(sizeof(double) * bead), *dN = (double *)malloc(sizeof(double) * bead);
    double s1 = orc_cv_com_distance(s, R, ga, na, gb, nb, d1);
    double sN = orc_cv_com_distance(s, R + bead * (size_t)(N - 1), ga, na, gb, nb, dN);
    double S = sN - s1, V = 0.0, dVdS = 0.0;
    for (int k = 0; k < nh; k++) {
        double u = (S - hills[k]) / sigma, e = w * exp(-0.5 * u * u);
        V += e;
        dVdS += -e * u / sigma;
    }
    if (grad_add) {
        memset(grad_add, 0, sizeof(double) * bead * (size_t)N);
        for (size_t o = 0; o < bead; o++) {
            grad_add[o] += -dVdS * d1[o];                          /* dS/dR^1 = -ds/dR^1 */
            grad_add[bead * (size_t)(N - 1) + o] += dVdS * dN[o];  /* dS/dR^N = +ds/dR^N */
        }
    }
    if (out) out[0] = S, out[1] = s1, out[2] = sN;
    free(d1), free(dN);
    return V;
}

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
