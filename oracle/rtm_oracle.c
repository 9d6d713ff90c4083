/*
 * rtm_oracle.c -- CPU ORACLE.  TEST INFRASTRUCTURE ONLY.
 *
 * A plain, slow, fp64 implementation of what the hot path of arxiv 2201.06914 computes:
 * time-domain FD wave propagation (acoustic 2D/3D, pseudo-acoustic TTI 2D/3D) with the
 * randomized-trace imaging condition accumulated in the time loop (Eq. 3),
 * the image (Eq. 3), the exact zero-lag image from stored history (Eq. 2, in the
 * u.v form -- reading C4 of DESIGN.md) and horizontal subsurface-offset volumes (Eq. 4,
 * PAPER.md:L49-52).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, load or call this file.  It shares no code with the CUDA path (paper_2201_06914_b200/):
 * no common header, table, helper or constant generator.  The product never falls back to it.
 *
 * The paper gives NO discretisation (no FD order, boundary, source/receiver handling, time step);
 * those follow SURVEY.md 8(c) O1-O7 / DESIGN.md "Readings".  Each function cites its passage.
 *
 * Arithmetic: fp64.  Inputs that the GPU receives in fp32 (coefficient arrays, damping tables,
 * FD weights, interpolation weights, wavelets, data, probes) are taken as the SAME fp32 bits and
 * promoted to fp64 (reading C18), so that the only GPU-vs-oracle difference is fp32 arithmetic.
 *
 * Pins (tests/test_oracle_*.py): Z = sqrt(nt) I  =>  image == exact image; Uz == history^T Z via
 * numpy matmul; estimator mean/variance closed form (Avron-Toledo); gather[h=0] == image, brute
 * force gather (scalar and vector offsets; spike pair at midpoint / half-offset); dot test <Fq,d> = <q,F^T d>; analytic 2D/3D Green's functions incl. 2nd-order
 * convergence in dt; TTI: H symmetric negative semi-definite, eps=delta=theta=0 => p == r ==
 * acoustic, theta -> theta+pi invariance; coefficient closed forms; two-field TTI probing (C29): central
 * differences of the misfit in K2 against sum_n (D p w_p + D r w_r) / (K2 h^2) from the histories.
 * Damped update (C7/C23): the centred scheme solved for the new level, stepped in numpy, to 1e-12 on the whole
 * padded grid; in-layer attenuation exp(-int sigma/c) of the stated profile.  TTI kinematics (C10): homogeneous
 * VTI is faster along x by sqrt(1 + 2 eps); with theta = +30 deg the fast direction is (cos th, -sin th).
 * 3D TTI (C30; tests/test_oracle_tti3d.py): dot test, H symmetric negative semi-definite, H_perp + H_par = Laplacian for
 * constant angles, eps = delta = 0 => p == r == acoustic, tilted kinematics (c along n, c sqrt(1+2 eps) along e1, e2).
 * Two probed fields in 3D (C29 + C30): 1/2 (Pz + Rz) == the one-field planes, PZ == hist^T Z by numpy per field, history
 * field 0 / 1 == physical part of the p / r snapshot.
 * PARITY UNPINNED (free choices no external fact fixes; the implementation is pinned to its stated design, the
 * design itself is a choice): the damping profile shape and strength, the wavelet delay, and imaging the single
 * TTI field (p+r)/2.
 *
 * Grid layout: physical grid n = (nx,[ny],nz), absorbing layer nb on every side, padded grid
 * P = n + 2 nb; zeros outside P (reading C8).  z is the contiguous axis.  Internally every field
 * lives on an extended grid E = P + 2*4 so that the order-8 stencil reads the zero exterior.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define HALO 4

typedef struct {
    int ndim;      /* 2 or 3 */
    int n[3];      /* physical points: 2D uses n[0]=nx, n[1]=nz ; 3D nx,ny,nz */
    int nb;        /* absorbing layer points on every side */
    int physics;   /* 0 acoustic, 1 TTI (2D: tilt theta; 3D: tilt theta and azimuth phi) */
    int nt;
    int r;
    double h;      /* grid spacing [m]; must be exactly representable as the fp32 the GPU gets */
    double dt;     /* time step [s] */
} orc_cfg;

/* ---- FD weights, rounded to fp32 (reading C18), textbook Fornberg order 8 ------------------ */
/* second derivative: w_1..w_4 ; the centre weight is DEFINED as w_0 = -2 sum_j w_j of the rounded
 * side weights, so that the discrete Laplacian annihilates constants exactly (reading C21).     */
static double W2(int j) {
    static const double w[5] = {0.0, 8.0 / 5.0, -1.0 / 5.0, 8.0 / 315.0, -1.0 / 560.0};
    return (double)(float)w[j];
}
/* centred first derivative (undivided: the 1/h^2 of two applications lives in K2, reading C22) */
static double W1(int j) {
    static const double c[5] = {0.0, 4.0 / 5.0, -1.0 / 5.0, 4.0 / 105.0, -1.0 / 280.0};
    return (double)(float)c[j];
}

/* ---- geometry helpers ----------------------------------------------------------------------- */
typedef struct {
    int nd;
    int n[3], P[3], E[3];   /* as 3 axes (x,y,z); for 2D the y axis has n=P=E=1 and no halo     */
    int ho[3];              /* halo per axis (4, or 0 for the dummy y axis)                      */
    long sx, sy;            /* strides on E (z stride 1)                                         */
    long NE, Np, N;
    int nb;
} geom;

static void make_geom(const orc_cfg *c, geom *g) {
    g->nd = c->ndim;
    g->nb = c->nb;
    if (c->ndim == 2) {
        g->n[0] = c->n[0]; g->n[1] = 1; g->n[2] = c->n[1];
    } else {
        g->n[0] = c->n[0]; g->n[1] = c->n[1]; g->n[2] = c->n[2];
    }
    for (int a = 0; a < 3; a++) {
        int active = !(c->ndim == 2 && a == 1);
        g->P[a] = active ? g->n[a] + 2 * c->nb : 1;
        g->ho[a] = active ? HALO : 0;
        g->E[a] = g->P[a] + 2 * g->ho[a];
    }
    g->sy = g->E[2];
    g->sx = (long)g->E[1] * g->E[2];
    g->NE = (long)g->E[0] * g->E[1] * g->E[2];
    g->Np = (long)g->P[0] * g->P[1] * g->P[2];
    g->N = (long)g->n[0] * g->n[1] * g->n[2];
}
/* index on E of padded-grid point (jx,jy,jz) */
static inline long eidx(const geom *g, int jx, int jy, int jz) {
    return (long)(jx + g->ho[0]) * g->sx + (long)(jy + g->ho[1]) * g->sy + (jz + g->ho[2]);
}
static inline long pidx(const geom *g, int jx, int jy, int jz) {
    return ((long)jx * g->P[1] + jy) * g->P[2] + jz;
}
static inline int layer_of(const geom *g, int a) { return (g->nd == 2 && a == 1) ? 0 : g->nb; }

/* ==== O1. Coefficients ====================================================
 * Scheme: (1/c^2)(u_tt + 2 sigma u_t) - Lap u = q, centred differences in time.
 *   padded model  : edge-replicate vp (eps, delta, theta) into the layer; v_max = max vp
 *   d_a(i) = max(0, nb - i, i - (P_a-1-nb)) ; phi(s) = s - sin(2 pi s)/(2 pi)
 *   sigma(i) = sigma_max * sum_a phi(d_a/nb) ; sigma_max = v_max ln(1000) / (nb h)
 *   damp_a[i] = sigma_max phi(d_a(i)/nb) dt            (per-axis tables, rounded to fp32)
 *   K2 = c^2 dt^2 / (h^2 (1 + sigma dt))               (rounded to fp32; acoustic AND TTI, C22)
 *   K1 = (1 - s)/(1 + s), s = sum_a damp_a[i_a]        (rebuilt from the fp32 tables, see K1())
 *   TTI: epsh = 1 + 2 eps ; delh = sqrt(1 + 2 min(delta, eps)) ; cos(theta), sin(theta)
 * Outputs: K2,epsh,delh,cosT,sinT [Np] canonical padded order; damp = concat over active axes.
 */
static int coeffs_impl(const orc_cfg *c, const float *vp, const float *eps, const float *delta,
               const float *theta, const float *phi, float *K2, float *damp, float *epsh, float *delh, float *cosT,
               float *sinT, float *cosP, float *sinP) {
    geom g; make_geom(c, &g);
    double vmax = 0.0;
    for (long i = 0; i < g.N; i++) if (vp[i] > vmax) vmax = vp[i];
    double smax = (c->nb > 0) ? vmax * log(1000.0) / ((double)c->nb * c->h) : 0.0;
    /* exact (unrounded) per-axis sigma_a * dt, and the fp32 tables */
    double *sd[3] = {0, 0, 0};
    long off = 0;
    for (int a = 0; a < 3; a++) {
        sd[a] = (double *)calloc((size_t)g.P[a], sizeof(double));
        if (g.nd == 2 && a == 1) continue;
        for (int i = 0; i < g.P[a]; i++) {
            int d = 0;
            if (c->nb - i > d) d = c->nb - i;
            if (i - (g.P[a] - 1 - c->nb) > d) d = i - (g.P[a] - 1 - c->nb);
            double s = (c->nb > 0) ? (double)d / (double)c->nb : 0.0;
            double phi = s - sin(2.0 * M_PI * s) / (2.0 * M_PI);
            sd[a][i] = smax * phi * c->dt;
            damp[off + i] = (float)sd[a][i];
        }
        off += g.P[a];
    }
    for (int jx = 0; jx < g.P[0]; jx++)
        for (int jy = 0; jy < g.P[1]; jy++)
            for (int jz = 0; jz < g.P[2]; jz++) {
                int ix = jx - layer_of(&g, 0), iy = jy - layer_of(&g, 1), iz = jz - layer_of(&g, 2);
                if (ix < 0) ix = 0; if (ix > g.n[0] - 1) ix = g.n[0] - 1;
                if (iy < 0) iy = 0; if (iy > g.n[1] - 1) iy = g.n[1] - 1;
                if (iz < 0) iz = 0; if (iz > g.n[2] - 1) iz = g.n[2] - 1;
                long src = ((long)ix * g.n[1] + iy) * g.n[2] + iz;
                long dst = pidx(&g, jx, jy, jz);
                double cc = vp[src];
                double sdt = sd[0][jx] + sd[1][jy] + sd[2][jz];
                K2[dst] = (float)(cc * cc * c->dt * c->dt / (c->h * c->h * (1.0 + sdt)));
                if (c->physics == 1) {
                    double e = eps[src], dl = delta[src], th = theta[src];
                    if (dl > e) dl = e;
                    epsh[dst] = (float)(1.0 + 2.0 * e);
                    delh[dst] = (float)sqrt(1.0 + 2.0 * dl);
                    cosT[dst] = (float)cos(th);
                    sinT[dst] = (float)sin(th);
                    if (phi) {          /* 3D: azimuth of the symmetry axis (reading C30) */
                        cosP[dst] = (float)cos((double)phi[src]);
                        sinP[dst] = (float)sin((double)phi[src]);
                    }
                }
            }
    for (int a = 0; a < 3; a++) free(sd[a]);
    return 0;
}

int orc_coeffs(const orc_cfg *c, const float *vp, const float *eps, const float *delta,
               const float *theta, float *K2, float *damp, float *epsh, float *delh, float *cosT,
               float *sinT) {
    return coeffs_impl(c, vp, eps, delta, theta, NULL, K2, damp, epsh, delh, cosT, sinT, NULL, NULL);
}
/* 3D TTI (reading C30): the same plus cos / sin of the azimuth phi of the symmetry axis */
int orc_coeffs3(const orc_cfg *c, const float *vp, const float *eps, const float *delta, const float *theta,
                const float *phi, float *K2, float *damp, float *epsh, float *delh, float *cosT, float *sinT,
                float *cosP, float *sinP) {
    return coeffs_impl(c, vp, eps, delta, theta, phi, K2, damp, epsh, delh, cosT, sinT, cosP, sinP);
}

/* K1 at padded point (jx,jy,jz) from the fp32 per-axis tables (O1) */
static inline double K1_at(const geom *g, const float *damp, int jx, int jy, int jz) {
    double s = (double)damp[jx];
    long off = g->P[0];
    if (g->nd == 3) { s += (double)damp[off + jy]; off += g->P[1]; }
    s += (double)damp[off + jz];
    return (1.0 - s) / (1.0 + s);
}

/* ==== Multilinear interpolation (reading C9) ==================================================
 * position x_a [m, fp32] -> f = x_a / h (fp64 division of the two fp32 values);
 * i0 = floor(f), clipped to n_a-2 so that the last grid point is reached with frac = 1;
 * weights (1-frac, frac) per axis; corner weight = product over axes, rounded to fp32.
 * Returns the number of corners (2^d), or -1 if the position is outside [0,(n_a-1)h].
 * idxE = index on E (for fields), idxN = index on the physical grid.                           */
static int corners(const orc_cfg *c, const geom *g, const float *xyz, long *idxE, double *w) {
    int i0[3] = {0, 0, 0};
    double fr[3] = {0, 0, 0};
    float hf = (float)c->h;
    for (int a = 0, k = 0; a < 3; a++) {
        if (g->nd == 2 && a == 1) continue;
        double f = (double)xyz[k++] / (double)hf;
        if (!(f >= 0.0) || f > (double)(g->n[a] - 1)) return -1;
        int i = (int)floor(f);
        if (i > g->n[a] - 2) i = g->n[a] - 2;
        if (i < 0) i = 0;
        i0[a] = i;
        fr[a] = f - (double)i;
    }
    int nc = 0;
    for (int bx = 0; bx < 2; bx++)
        for (int by = 0; by < 2; by++)
            for (int bz = 0; bz < 2; bz++) {
                if (g->nd == 2 && by == 1) continue;
                if ((bx && g->n[0] == 1) || (by && g->n[1] == 1) || (bz && g->n[2] == 1)) {
                    idxE[nc] = 0; w[nc++] = 0.0; continue;
                }
                double ww = (bx ? fr[0] : 1.0 - fr[0]);
                if (g->nd == 3) ww *= (by ? fr[1] : 1.0 - fr[1]);
                ww *= (bz ? fr[2] : 1.0 - fr[2]);
                idxE[nc] = eidx(g, i0[0] + bx + layer_of(g, 0), i0[1] + by + layer_of(g, 1),
                                i0[2] + bz + layer_of(g, 2));
                w[nc++] = (double)(float)ww;
            }
    return nc;
}

/* ==== Spatial operators ======================================================================= */
/* Order-8 Laplacian in difference form, sum_axes sum_j w_j (u[+j] - 2u + u[-j])  (O2, C21);
 * undivided: 1/h^2 is inside K2.                                                                */
static inline double lap8(const geom *g, const double *u, long i) {
    double L = 0.0;
    for (int j = 1; j <= 4; j++) {
        double s = (u[i + j * g->sx] - 2.0 * u[i] + u[i - j * g->sx]) +
                   (u[i + j] - 2.0 * u[i] + u[i - j]);
        if (g->nd == 3) s += (u[i + j * g->sy] - 2.0 * u[i] + u[i - j * g->sy]);
        L += W2(j) * s;
    }
    return L;
}
/* undivided centred first derivatives, order 8 */
static inline double dx8(const geom *g, const double *f, long i) {
    double s = 0.0;
    for (int j = 1; j <= 4; j++) s += W1(j) * (f[i + j * g->sx] - f[i - j * g->sx]);
    return s;
}
static inline double dz8(const double *f, long i) {
    double s = 0.0;
    for (int j = 1; j <= 4; j++) s += W1(j) * (f[i + j] - f[i - j]);
    return s;
}

static inline double dy8(const geom *g, const double *f, long i) {
    double s = 0.0;
    for (int j = 1; j <= 4; j++) s += W1(j) * (f[i + j * g->sy] - f[i - j * g->sy]);
    return s;
}

/* Rotated self-adjoint operators in 3D (reading C30; "TTI", L81 "generalize to 3D").  Symmetry axis
 *   n  = (sin th cos ph, sin th sin ph, cos th)            (tilt th from the z axis, azimuth ph from the x axis)
 * and an orthonormal basis of the plane perpendicular to it
 *   e1 = (cos th cos ph, cos th sin ph, -sin th),   e2 = (-sin ph, cos ph, 0).
 * With G_v f = v . (Dx f, Dy f, Dz f)  (undivided centred order-8 first derivatives, evaluated on P, zero outside):
 *   which = 1:  H_par  f = -G_n^T G_n f              = Dx(nx g) + Dy(ny g) + Dz(nz g),          g = G_n f
 *   which = 0:  H_perp f = -(G_e1^T G_e1 + G_e2^T G_e2) f = Dx(e1x g1 + e2x g2) + Dy(e1y g1 + e2y g2) + Dz(e1z g1),
 *                                                                                    g1 = G_e1 f, g2 = G_e2 f
 * (D^T = -D with zeros outside P, reading C8).  For ph = 0 and fields that do not depend on y this is the 2D pair
 * above; for constant angles H_perp + H_par = Dx Dx + Dy Dy + Dz Dz exactly (e1, e2, n orthonormal).
 * f, out, t1, t2, t3 live on E; ct, st, cp, sp are [Np] fp32.                                              */
static void tti_H3(const geom *g, const float *ct, const float *st, const float *cp, const float *sp, int which,
                   const double *f, double *out, double *t1, double *t2, double *t3) {
    memset(t1, 0, (size_t)g->NE * sizeof(double));
    memset(t2, 0, (size_t)g->NE * sizeof(double));
    memset(t3, 0, (size_t)g->NE * sizeof(double));
#pragma omp parallel for schedule(static)
    for (int jx = 0; jx < g->P[0]; jx++)
        for (int jy = 0; jy < g->P[1]; jy++)
            for (int jz = 0; jz < g->P[2]; jz++) {
                long i = eidx(g, jx, jy, jz);
                long p = pidx(g, jx, jy, jz);
                double cT = ct[p], sT = st[p], cP = cp[p], sP = sp[p];
                double fx = dx8(g, f, i), fy = dy8(g, f, i), fz = dz8(f, i);
                if (which == 1) {
                    double nx = sT * cP, ny = sT * sP, nz = cT;
                    double gg = nx * fx + ny * fy + nz * fz;
                    t1[i] = nx * gg; t2[i] = ny * gg; t3[i] = nz * gg;
                } else {
                    double e1x = cT * cP, e1y = cT * sP, e1z = -sT, e2x = -sP, e2y = cP;
                    double g1 = e1x * fx + e1y * fy + e1z * fz;
                    double g2 = e2x * fx + e2y * fy;
                    t1[i] = e1x * g1 + e2x * g2; t2[i] = e1y * g1 + e2y * g2; t3[i] = e1z * g1;
                }
            }
#pragma omp parallel for schedule(static)
    for (int jx = 0; jx < g->P[0]; jx++)
        for (int jy = 0; jy < g->P[1]; jy++)
            for (int jz = 0; jz < g->P[2]; jz++) {
                long i = eidx(g, jx, jy, jz);
                out[i] = dx8(g, t1, i) + dy8(g, t2, i) + dz8(t3, i);
            }
}

/* test hook: apply the 3D H_perp / H_par to a padded-grid function (pins: symmetry, definiteness, rotation invariance) */
int orc_tti_H3(const orc_cfg *c, const float *cosT, const float *sinT, const float *cosP, const float *sinP, int which,
               const double *fP, double *outP) {
    geom g; make_geom(c, &g);
    if (c->ndim != 3) return -1;
    double *f = calloc((size_t)g.NE, sizeof(double)), *o = calloc((size_t)g.NE, sizeof(double));
    double *t1 = malloc((size_t)g.NE * sizeof(double)), *t2 = malloc((size_t)g.NE * sizeof(double)), *t3 = malloc((size_t)g.NE * sizeof(double));
    for (int jx = 0; jx < g.P[0]; jx++)
        for (int jy = 0; jy < g.P[1]; jy++)
            for (int jz = 0; jz < g.P[2]; jz++) f[eidx(&g, jx, jy, jz)] = fP[pidx(&g, jx, jy, jz)];
    tti_H3(&g, cosT, sinT, cosP, sinP, which, f, o, t1, t2, t3);
    for (int jx = 0; jx < g.P[0]; jx++)
        for (int jy = 0; jy < g.P[1]; jy++)
            for (int jz = 0; jz < g.P[2]; jz++) outP[pidx(&g, jx, jy, jz)] = o[eidx(&g, jx, jy, jz)];
    free(f); free(o); free(t1); free(t2); free(t3);
    return 0;
}

/* Rotated self-adjoint operators of O5 (2D; symmetry axis (sin th, cos th) in (x,z)):
 *   which = 0:  H_perp f = Dx(cos g) - Dz(sin g),  g = cos Dx f - sin Dz f      (= -G^T G f)
 *   which = 1:  H_par  f = Dx(sin g) + Dz(cos g),  g = sin Dx f + cos Dz f
 * g is evaluated on P only and is zero outside (so that D^T = -D, reading C8).
 * f, out, t1, t2 live on E; ct, st are [Np] fp32.                                               */
static void tti_H(const geom *g, const float *ct, const float *st, int which, const double *f,
                  double *out, double *t1, double *t2) {
    memset(t1, 0, (size_t)g->NE * sizeof(double));
    memset(t2, 0, (size_t)g->NE * sizeof(double));
#pragma omp parallel for schedule(static)
    for (int jx = 0; jx < g->P[0]; jx++)
        for (int jz = 0; jz < g->P[2]; jz++) {
            long i = eidx(g, jx, 0, jz);
            long p = pidx(g, jx, 0, jz);
            double cs = ct[p], sn = st[p];
            double fx = dx8(g, f, i), fz = dz8(f, i);
            if (which == 0) {
                double gg = cs * fx - sn * fz;
                t1[i] = cs * gg;   /* enters Dx */
                t2[i] = sn * gg;   /* enters Dz */
            } else {
                double gg = sn * fx + cs * fz;
                t1[i] = sn * gg;
                t2[i] = cs * gg;
            }
        }
#pragma omp parallel for schedule(static)
    for (int jx = 0; jx < g->P[0]; jx++)
        for (int jz = 0; jz < g->P[2]; jz++) {
            long i = eidx(g, jx, 0, jz);
            out[i] = (which == 0) ? dx8(g, t1, i) - dz8(t2, i) : dx8(g, t1, i) + dz8(t2, i);
        }
}

/* test hook: apply H_perp / H_par to a padded-grid function (pins: symmetry, definiteness) */
int orc_tti_H(const orc_cfg *c, const float *cosT, const float *sinT, int which, const double *fP,
              double *outP) {
    geom g; make_geom(c, &g);
    if (c->ndim != 2) return -1;
    double *f = calloc((size_t)g.NE, sizeof(double)), *o = calloc((size_t)g.NE, sizeof(double));
    double *t1 = malloc((size_t)g.NE * sizeof(double)), *t2 = malloc((size_t)g.NE * sizeof(double));
    for (int jx = 0; jx < g.P[0]; jx++)
        for (int jz = 0; jz < g.P[2]; jz++) f[eidx(&g, jx, 0, jz)] = fP[pidx(&g, jx, 0, jz)];
    tti_H(&g, cosT, sinT, which, f, o, t1, t2);
    for (int jx = 0; jx < g.P[0]; jx++)
        for (int jz = 0; jz < g.P[2]; jz++) outP[pidx(&g, jx, 0, jz)] = o[eidx(&g, jx, 0, jz)];
    free(f); free(o); free(t1); free(t2);
    return 0;
}

/* ==== O2/O3/O5/O6. One propagation pass with fused probing ====================================
 * adjoint = 0 (O2, O5): n = 0..nt-1,  inject  K2 h^(2-d) w val[n][s]   at inj points,
 *                       sample  sum_c w new[c]                          at smp points.
 * adjoint = 1 (O3, O6): n = nt-1..0,  inject  K2 h^2 w val[n][j]        (TTI: 1/2 into p and r),
 *                       sample  h^(-d) sum_c w new[c]                   (TTI: w_p + w_r).
 * Step n:  new = cur + K1 (cur - prev) + K2 * Op(cur)        for every point of P
 *          inject row n ; sample row n ; probe: PZ[k][x] += Z[n][k] * new[x] (physical x only,
 *          PAPER.md:L45-47 Eq. 3 with reading C6: row n probes the newly computed field);
 *          hist[n] = new (physical grid) ; rotate prev <- cur <- new.
 * TTI forward:  p_new = .. + K2 (epsh A + delh B), r_new = .. + K2 (delh A + B),
 *               A = H_perp p, B = H_par r;  sampled / probed field = (p_new + r_new)/2.
 * TTI adjoint:  a = epsh p + delh r, b = delh p + r, p_new = .. + K2 H_perp a, r_new = .. + K2 H_par b.
 * snaps: [nsnap][nf][Np] (nf = 1 acoustic, 2 TTI), the field(s) right after step snap_steps[i]
 * (including that step's injection).
 * Returns 0, or -2 if a position is outside the physical grid.                                   */
static int propagate(const orc_cfg *c, int adjoint, const float *K2, const float *damp,
                  const float *epsh, const float *delh, const float *cosT, const float *sinT,
                  const float *cosP, const float *sinP /* 3D TTI only, else NULL */,
                  int ninj, const float *inj_xyz, const float *inj_val /*[nt][ninj]*/,
                  int nsmp, const float *smp_xyz, double *smp_out /*[nt][nsmp] or NULL*/,
                  const float *Z /*[nt][r] or NULL*/, double *PZ /*[np][r][N] or NULL*/,
                  double *hist /*[nt][np][N] or NULL*/, int nsnap, const int *snap_steps,
                  double *snaps, int np /* probed fields: 1, or 2 = p and r apart (TTI) */) {
    geom g; make_geom(c, &g);
    const int d = c->ndim, tti = (c->physics == 1);
    if (tti && d == 3 && (!cosP || !sinP)) return -1;
    if (np != 1 && !(np == 2 && tti)) return -1;
    const int nf = tti ? 2 : 1;
    const int nc = 1 << d;

    /* interpolation tables */
    long *iE = malloc(sizeof(long) * (size_t)(ninj > 0 ? ninj : 1) * 8);
    double *iW = malloc(sizeof(double) * (size_t)(ninj > 0 ? ninj : 1) * 8);
    long *sE = malloc(sizeof(long) * (size_t)(nsmp > 0 ? nsmp : 1) * 8);
    double *sW = malloc(sizeof(double) * (size_t)(nsmp > 0 ? nsmp : 1) * 8);
    int bad = 0;
    for (int s = 0; s < ninj; s++) if (corners(c, &g, inj_xyz + (long)s * d, iE + 8L * s, iW + 8L * s) < 0) bad = 1;
    for (int s = 0; s < nsmp; s++) if (corners(c, &g, smp_xyz + (long)s * d, sE + 8L * s, sW + 8L * s) < 0) bad = 1;
    if (bad) { free(iE); free(iW); free(sE); free(sW); return -2; }

    /* map E-index -> padded canonical index for K2 lookups at injection corners */
    double inj_scale = adjoint ? c->h * c->h : pow(c->h, 2.0 - d);
    double smp_scale = adjoint ? pow(c->h, -(double)d) : 1.0;
    if (tti) { if (adjoint) inj_scale *= 0.5; else smp_scale *= 0.5; }

    double *F[2][3];          /* [field][prev,cur,new] on E */
    for (int f = 0; f < 2; f++) for (int k = 0; k < 3; k++)
        F[f][k] = (f < nf) ? calloc((size_t)g.NE, sizeof(double)) : NULL;
    double *A = NULL, *B = NULL, *t1 = NULL, *t2 = NULL, *t3 = NULL, *ma = NULL, *mb = NULL;
    if (tti) {
        A = calloc((size_t)g.NE, sizeof(double)); B = calloc((size_t)g.NE, sizeof(double));
        t1 = malloc((size_t)g.NE * sizeof(double)); t2 = malloc((size_t)g.NE * sizeof(double));
        t3 = malloc((size_t)g.NE * sizeof(double));
        ma = calloc((size_t)g.NE, sizeof(double)); mb = calloc((size_t)g.NE, sizeof(double));
    }
    if (PZ) memset(PZ, 0, sizeof(double) * (size_t)np * (size_t)c->r * (size_t)g.N);

    for (int step = 0; step < c->nt; step++) {
        const int n = adjoint ? c->nt - 1 - step : step;
        double *pp = F[0][0], *pc = F[0][1], *pn = F[0][2];
        double *rp = F[1][0], *rc = F[1][1], *rn = F[1][2];
        if (!tti) {
#pragma omp parallel for schedule(static)
            for (int jx = 0; jx < g.P[0]; jx++)
                for (int jy = 0; jy < g.P[1]; jy++)
                    for (int jz = 0; jz < g.P[2]; jz++) {
                        long i = eidx(&g, jx, jy, jz);
                        double k1 = K1_at(&g, damp, jx, jy, jz);
                        double k2 = K2[pidx(&g, jx, jy, jz)];
                        pn[i] = pc[i] + k1 * (pc[i] - pp[i]) + k2 * lap8(&g, pc, i);
                    }
        } else {
            const double *opA = pc, *opB = rc;
            if (adjoint) {     /* pre-mix (O6) */
#pragma omp parallel for schedule(static)
                for (int jx = 0; jx < g.P[0]; jx++)
                    for (int jy = 0; jy < g.P[1]; jy++)
                    for (int jz = 0; jz < g.P[2]; jz++) {
                        long i = eidx(&g, jx, jy, jz), p = pidx(&g, jx, jy, jz);
                        ma[i] = (double)epsh[p] * pc[i] + (double)delh[p] * rc[i];
                        mb[i] = (double)delh[p] * pc[i] + rc[i];
                    }
                opA = ma; opB = mb;
            }
            if (d == 2) {
                tti_H(&g, cosT, sinT, 0, opA, A, t1, t2);
                tti_H(&g, cosT, sinT, 1, opB, B, t1, t2);
            } else {
                tti_H3(&g, cosT, sinT, cosP, sinP, 0, opA, A, t1, t2, t3);
                tti_H3(&g, cosT, sinT, cosP, sinP, 1, opB, B, t1, t2, t3);
            }
#pragma omp parallel for schedule(static)
            for (int jx = 0; jx < g.P[0]; jx++)
                for (int jy = 0; jy < g.P[1]; jy++)
                for (int jz = 0; jz < g.P[2]; jz++) {
                    long i = eidx(&g, jx, jy, jz), p = pidx(&g, jx, jy, jz);
                    double k1 = K1_at(&g, damp, jx, jy, jz), k2 = K2[p];
                    double e = epsh[p], dl = delh[p];
                    double ra = adjoint ? A[i] : e * A[i] + dl * B[i];    /* post-mix (O5) */
                    double rb = adjoint ? B[i] : dl * A[i] + B[i];
                    pn[i] = pc[i] + k1 * (pc[i] - pp[i]) + k2 * ra;
                    rn[i] = rc[i] + k1 * (rc[i] - rp[i]) + k2 * rb;
                }
        }
        /* inject row n (a3): new[corner] += K2[corner] * scale * w * val */
        for (int s = 0; s < ninj; s++)
            for (int k = 0; k < nc; k++) {
                double w = iW[8L * s + k];
                if (w == 0.0) continue;
                long i = iE[8L * s + k];
                /* recover padded coordinates of i to look K2 up */
                long jx = i / g.sx - g.ho[0], rem = i % g.sx;
                long jy = rem / g.sy - g.ho[1], jz = rem % g.sy - g.ho[2];
                double k2 = K2[pidx(&g, (int)jx, (int)jy, (int)jz)];
                double v = k2 * inj_scale * w * (double)inj_val[(long)n * ninj + s];
                pn[i] += v;
                if (tti) rn[i] += v;
            }
        /* sample row n (a4) */
        if (smp_out)
            for (int s = 0; s < nsmp; s++) {
                double acc = 0.0;
                for (int k = 0; k < nc; k++) {
                    double w = sW[8L * s + k];
                    if (w == 0.0) continue;
                    long i = sE[8L * s + k];
                    acc += w * (tti ? pn[i] + rn[i] : pn[i]);
                }
                smp_out[(long)n * nsmp + s] = smp_scale * acc;
            }
        /* probe (a5) and history on the physical grid */
        if (PZ || hist) {
#pragma omp parallel for schedule(static)
            for (int ix = 0; ix < g.n[0]; ix++)
                for (int iy = 0; iy < g.n[1]; iy++)
                    for (int iz = 0; iz < g.n[2]; iz++) {
                        long i = eidx(&g, ix + layer_of(&g, 0), iy + layer_of(&g, 1), iz + layer_of(&g, 2));
                        long x = ((long)ix * g.n[1] + iy) * g.n[2] + iz;
                        for (int f = 0; f < np; f++) {
                            /* one probed field 1/2 (p + r) (reading C10), or p and r apart (reading C29) */
                            double u = np == 2 ? (f ? rn[i] : pn[i]) : (tti ? 0.5 * (pn[i] + rn[i]) : pn[i]);
                            if (hist) hist[((long)n * np + f) * g.N + x] = u;
                            if (PZ && Z)
                                for (int k = 0; k < c->r; k++)
                                    PZ[((long)f * c->r + k) * g.N + x] += (double)Z[(long)n * c->r + k] * u;
                        }
                    }
        }
        for (int q = 0; q < nsnap; q++)
            if (snap_steps[q] == n)
                for (int f = 0; f < nf; f++)
                    for (int jx = 0; jx < g.P[0]; jx++)
                        for (int jy = 0; jy < g.P[1]; jy++)
                            for (int jz = 0; jz < g.P[2]; jz++)
                                snaps[((long)q * nf + f) * g.Np + pidx(&g, jx, jy, jz)] =
                                    F[f][2][eidx(&g, jx, jy, jz)];
        /* rotate */
        for (int f = 0; f < nf; f++) {
            double *t = F[f][0]; F[f][0] = F[f][1]; F[f][1] = F[f][2]; F[f][2] = t;
        }
    }
    for (int f = 0; f < 2; f++) for (int k = 0; k < 3; k++) free(F[f][k]);
    free(A); free(B); free(t1); free(t2); free(t3); free(ma); free(mb);
    free(iE); free(iW); free(sE); free(sW);
    return 0;
}

int orc_propagate(const orc_cfg *c, int adjoint, const float *K2, const float *damp,
                  const float *epsh, const float *delh, const float *cosT, const float *sinT,
                  int ninj, const float *inj_xyz, const float *inj_val, int nsmp, const float *smp_xyz,
                  double *smp_out, const float *Z, double *PZ /*[r][N]*/, double *hist /*[nt][N]*/, int nsnap,
                  const int *snap_steps, double *snaps) {
    return propagate(c, adjoint, K2, damp, epsh, delh, cosT, sinT, NULL, NULL, ninj, inj_xyz, inj_val, nsmp, smp_xyz, smp_out,
                     Z, PZ, hist, nsnap, snap_steps, snaps, 1);
}

/* 3D pseudo-acoustic TTI (reading C30): the same pass with the rotated operators tti_H3 (tilt and azimuth).        */
int orc_propagate3(const orc_cfg *c, int adjoint, const float *K2, const float *damp,
                   const float *epsh, const float *delh, const float *cosT, const float *sinT, const float *cosP,
                   const float *sinP, int ninj, const float *inj_xyz, const float *inj_val, int nsmp,
                   const float *smp_xyz, double *smp_out, const float *Z, double *PZ /*[r][N]*/, double *hist /*[nt][N]*/,
                   int nsnap, const int *snap_steps, double *snaps) {
    return propagate(c, adjoint, K2, damp, epsh, delh, cosT, sinT, cosP, sinP, ninj, inj_xyz, inj_val, nsmp, smp_xyz,
                     smp_out, Z, PZ, hist, nsnap, snap_steps, snaps, 1);
}

/* Four compressed arrays for the TTI gradient (Eq. 2-3 applied to the coupled (p, r) system of
 * PAPER.md:L77, reading C29): the same pass, but p and r are probed apart,
 * PZ [2][r][N] = (Pz, Rz) forward / (Wpz, Wrz) adjoint, hist [nt][2][N].  Eq. 3 over the 2r planes,
 * (1/r) sum_k (Pz_k Wpz_k + Rz_k Wrz_k), then estimates sum_t (p w_p + r w_r).                            */
int orc_propagate_pr(const orc_cfg *c, int adjoint, const float *K2, const float *damp,
                     const float *epsh, const float *delh, const float *cosT, const float *sinT,
                     int ninj, const float *inj_xyz, const float *inj_val, int nsmp, const float *smp_xyz,
                     double *smp_out, const float *Z, double *PZ /*[2][r][N]*/, double *hist /*[nt][2][N]*/,
                     int nsnap, const int *snap_steps, double *snaps) {
    return propagate(c, adjoint, K2, damp, epsh, delh, cosT, sinT, NULL, NULL, ninj, inj_xyz, inj_val, nsmp, smp_xyz, smp_out,
                     Z, PZ, hist, nsnap, snap_steps, snaps, 2);
}

/* The same four arrays for 3D TTI (readings C29 + C30: Eq. 2-3, on the (p, r) system of L77 in the 3D
 * form of L81): orc_propagate3 with p and r probed apart, PZ [2][r][N], hist [nt][2][N].                        */
int orc_propagate3_pr(const orc_cfg *c, int adjoint, const float *K2, const float *damp,
                      const float *epsh, const float *delh, const float *cosT, const float *sinT, const float *cosP,
                      const float *sinP, int ninj, const float *inj_xyz, const float *inj_val, int nsmp,
                      const float *smp_xyz, double *smp_out, const float *Z, double *PZ /*[2][r][N]*/,
                      double *hist /*[nt][2][N]*/, int nsnap, const int *snap_steps, double *snaps) {
    return propagate(c, adjoint, K2, damp, epsh, delh, cosT, sinT, cosP, sinP, ninj, inj_xyz, inj_val, nsmp, smp_xyz,
                     smp_out, Z, PZ, hist, nsnap, snap_steps, snaps, 2);
}

/* ==== O4. Images ============================================================================== */
/* Eq. 3: I[x] = scale * sum_k Uz[k][x] Vz[k][x], scale = 1/r                      */
void orc_image(int r, long N, const double *Uz, const double *Vz, double scale, double *I) {
    for (long x = 0; x < N; x++) {
        double s = 0.0;
        for (int k = 0; k < r; k++) s += Uz[(long)k * N + x] * Vz[(long)k * N + x];
        I[x] = scale * s;
    }
}
/* Eq. 2 in the u.v form (reading C4/C5): I[x] = sum_n uh[n][x] vh[n][x]           */
void orc_exact_image(int nt, long N, const double *uh, const double *vh, double *I) {
    for (long x = 0; x < N; x++) {
        double s = 0.0;
        for (int n = 0; n < nt; n++) s += uh[(long)n * N + x] * vh[(long)n * N + x];
        I[x] = s;
    }
}
/* Eq. 4, reading C11: offsets are integer grid points along x;
 * G[ih][x] = scale * sum_k Uz[k][x + h e_x] Vz[k][x - h e_x]; zero when x+h or x-h leaves [0,nx) */
void orc_offset_gather(int nx, long nrest /* ny*nz */, int r, const double *Uz, const double *Vz,
                       int nh, const int *offs, double scale, double *G) {
    long N = (long)nx * nrest;
    for (int ih = 0; ih < nh; ih++) {
        int h = offs[ih];
        for (int ix = 0; ix < nx; ix++)
            for (long q = 0; q < nrest; q++) {
                double s = 0.0;
                int a = ix + h, b = ix - h;
                if (a >= 0 && a < nx && b >= 0 && b < nx)
                    for (int k = 0; k < r; k++)
                        s += Uz[(long)k * N + (long)a * nrest + q] * Vz[(long)k * N + (long)b * nrest + q];
                G[(long)ih * N + (long)ix * nrest + q] = scale * s;
            }
    }
}

/* Eq. 4 with a VECTOR horizontal offset h = (hx, hy) in grid points (
 * PAPER.md:L81 "generalize to 3D"; reading C28): 3D grids [nx][ny][nz],
 * G[ih][x] = scale * sum_k Uz[k][x + hx e_x + hy e_y] Vz[k][x - hx e_x - hy e_y];
 * zero when either shifted point leaves [0,nx) x [0,ny).  offs = [nh][2] = (hx, hy) pairs.         */
void orc_offset_gather_xy(int nx, int ny, int nz, int r, const double *Uz, const double *Vz, int nh,
                          const int *offs, double scale, double *G) {
    long N = (long)nx * ny * nz;
    for (int ih = 0; ih < nh; ih++) {
        int hx = offs[2 * ih], hy = offs[2 * ih + 1];
        for (int ix = 0; ix < nx; ix++)
            for (int iy = 0; iy < ny; iy++)
                for (int iz = 0; iz < nz; iz++) {
                    int ax = ix + hx, ay = iy + hy, bx = ix - hx, by = iy - hy;
                    double s = 0.0;
                    if (ax >= 0 && ax < nx && ay >= 0 && ay < ny && bx >= 0 && bx < nx && by >= 0 && by < ny)
                        for (int k = 0; k < r; k++)
                            s += Uz[(long)k * N + ((long)ax * ny + ay) * nz + iz] *
                                 Vz[(long)k * N + ((long)bx * ny + by) * nz + iz];
                    G[(long)ih * N + ((long)ix * ny + iy) * nz + iz] = scale * s;
                }
    }
}

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
