/*
 * dock_oracle.c -- CPU ORACLE (double precision, plain C) for the DSDP docking-stage hot path.
 * TEST INFRASTRUCTURE ONLY: see the header of dock_oracle.h for who may call this, the
 * passages of PAPER.md each function follows, and which parts are "parity unpinned".
 *
 * No blocking, no lookup tables, no cell lists, no fusion: every function is the definition
 * or the algorithm written out in the paper's order.  OpenMP is used only ACROSS independent
 * poses / copies / grid nodes (never inside one evaluation), so results do not depend on the
 * number of threads.
 */
#include "dock_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define PI 3.14159265358979323846

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ---------------------------------------------------------------------------------------
 * Parameters: readings S1 (weights), S2 (XS radii and flags), S3, S7, S12, S14, S15, S19 of
 * SURVEY.md 8(c).  The paper prints none of them (PAPER.md:49 only says "same scoring
 * function" as Vina); they are inputs, so parity does not depend on the values.
 * ------------------------------------------------------------------------------------- */
void orc_default_params(orc_params *p)
{
    /* id order: C_H C_P N_P N_D N_A N_DA O_P O_D O_A O_DA S_P P_P F_H Cl_H Br_H I_H Met_D */
    static const double rad[17] = {1.9, 1.9, 1.8, 1.8, 1.8, 1.8, 1.7, 1.7, 1.7, 1.7,
                                   2.0, 2.1, 1.5, 1.8, 2.0, 2.2, 1.2};
    static const int hyd[17] = {1, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 1, 1, 1, 1, 0};
    static const int don[17] = {0, 0, 0, 1, 0, 1, 0, 1, 0, 1, 0, 0, 0, 0, 0, 0, 1};
    static const int acc[17] = {0, 0, 0, 0, 1, 1, 0, 0, 1, 1, 0, 0, 0, 0, 0, 0, 0};
    memset(p, 0, sizeof(*p));
    p->n_types = 17;
    for (int i = 0; i < 17; ++i) {
        p->radius[i] = rad[i];
        p->hydrophobic[i] = hyd[i];
        p->donor[i] = don[i];
        p->acceptor[i] = acc[i];
    }
    p->w[0] = -0.0356;
    p->w[1] = -0.00516;
    p->w[2] = 0.840;
    p->w[3] = -0.0351;
    p->w[4] = -0.587;
    p->cutoff = 8.0;
    p->k_wall = 10.0;
    p->t_mc = 1.2;
    p->amp_trans = 2.0;
    p->amp_rot = 0.3;
    p->bfgs_c1 = 1e-4;
    p->bfgs_shrink = 0.5;
    p->bfgs_max_trials = 12;
    p->bfgs_gtol = 1e-3;
    p->bfgs_curv_eps = 1e-8;
    p->cluster_rmsd = 2.0;
    p->topk = 10;
    p->optimizer = 0;
    p->bb_step = 1.0;
    p->bb_fallback = 0.1;
}

/* ---------------------------------------------------------------------------------------
 * O1 pair potential on surface distance d = r - R1 - R2 (terms named in
 * BASELINE.json:north_star).  Direct evaluation, no radial table.
 *   f = w1 exp(-(d/0.5)^2) + w2 exp(-((d-3)/2)^2) + w3 (d<0 ? d^2 : 0)
 *     + w4 [both hydrophobic] H(d) + w5 [donor-acceptor] B(d)
 *   H = 1 (d<0.5), 1.5-d (0.5<=d<1.5), 0 (d>=1.5);  B = 1 (d<-0.7), -d/0.7 (-0.7<=d<0), 0 (d>=0)
 * ------------------------------------------------------------------------------------- */
static int is_hbond_pair(const orc_params *p, int t1, int t2)
{
    return (p->donor[t1] && p->acceptor[t2]) || (p->donor[t2] && p->acceptor[t1]);
}

double orc_pair(const orc_params *p, int t1, int t2, double r, double *dfdr)
{
    double e = 0.0, de = 0.0;
    if (r < p->cutoff) {
        double d = r - p->radius[t1] - p->radius[t2];
        double a = d / 0.5;
        double g1 = exp(-a * a);
        e += p->w[0] * g1;
        de += p->w[0] * g1 * (-2.0 * a / 0.5);
        double b = (d - 3.0) / 2.0;
        double g2 = exp(-b * b);
        e += p->w[1] * g2;
        de += p->w[1] * g2 * (-2.0 * b / 2.0);
        if (d < 0.0) {
            e += p->w[2] * d * d;
            de += p->w[2] * 2.0 * d;
        }
        if (p->hydrophobic[t1] && p->hydrophobic[t2]) {
            if (d < 0.5) {
                e += p->w[3];
            } else if (d < 1.5) {
                e += p->w[3] * (1.5 - d);
                de += -p->w[3];
            }
        }
        if (is_hbond_pair(p, t1, t2)) {
            if (d < -0.7) {
                e += p->w[4];
            } else if (d < 0.0) {
                e += p->w[4] * (-d / 0.7);
                de += -p->w[4] / 0.7;
            }
        }
    }
    if (dfdr) *dfdr = de;
    return e;
}

/* distance of d to the nearest derivative kink of the ACTIVE piecewise-linear terms */
static double pair_kink_margin(const orc_params *p, int t1, int t2, double r)
{
    double m = fabs(r - p->cutoff);
    double d = r - p->radius[t1] - p->radius[t2];
    if (p->hydrophobic[t1] && p->hydrophobic[t2]) {
        m = fmin(m, fabs(d - 0.5));
        m = fmin(m, fabs(d - 1.5));
    }
    if (is_hbond_pair(p, t1, t2)) {
        m = fmin(m, fabs(d + 0.7));
        m = fmin(m, fabs(d));
    }
    return m;
}

/* ---------------------------------------------------------------------------------------
 * Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11), R-rules of SURVEY.md 8(c).
 * ------------------------------------------------------------------------------------- */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* counter = (copy, step, slot, system); key = (seed lo, seed hi) */
static void draw(uint64_t seed, uint32_t system, uint32_t copy, uint32_t step, uint32_t slot, uint32_t r[4])
{
    uint32_t ctr[4] = {copy, step, slot, system};
    uint32_t key[2] = {(uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32)};
    orc_philox4x32_10(ctr, key, r);
}

/* u = (r >> 8) * 2^-24, exact in fp32 and fp64 */
static double u24(uint32_t r) { return (double)(r >> 8) * (1.0 / 16777216.0); }

/* ---------------------------------------------------------------------------------------
 * O2 grid maps (eq. 2's inner sum at 198-199).
 * ------------------------------------------------------------------------------------- */
void orc_grid_geometry(const double center[3], const double size[3], double h, int dims[3], double origin[3])
{
    for (int c = 0; c < 3; ++c) {
        dims[c] = (int)floor(size[c] / h + 0.5) + 1;
        /* DESIGN.md reading D-ORG: the origin is rounded ONCE to fp32 so that both
         * implementations place node 0 at the same representable coordinate. */
        origin[c] = (double)(float)(center[c] - 0.5 * size[c]);
    }
}

void orc_build_grid(const orc_params *p, int np, const double *pxyz, const int32_t *ptype,
                    const int dims[3], const double origin[3], double h,
                    int n_lig_types, const int32_t *lig_types, double *G)
{
    const int nx = dims[0], ny = dims[1], nz = dims[2];
    const int64_t nodes = (int64_t)nx * ny * nz;
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t m = 0; m < nodes; ++m) {
        int ix = (int)(m % nx), iy = (int)((m / nx) % ny), iz = (int)(m / ((int64_t)nx * ny));
        double mx = origin[0] + h * ix, my = origin[1] + h * iy, mz = origin[2] + h * iz;
        for (int t = 0; t < n_lig_types; ++t) G[(int64_t)t * nodes + m] = 0.0;
        for (int j = 0; j < np; ++j) {
            double dx = mx - pxyz[3 * j], dy = my - pxyz[3 * j + 1], dz = mz - pxyz[3 * j + 2];
            double r = sqrt(dx * dx + dy * dy + dz * dz);
            if (!(r < p->cutoff)) continue;                    /* S3: strict, decided in double */
            for (int t = 0; t < n_lig_types; ++t)
                G[(int64_t)t * nodes + m] += orc_pair(p, lig_types[t], ptype[j], r, NULL);
        }
    }
}

/* Diagnostic only (changes no result): flags[node] = 1 iff some protein atom lies within `margin` of the cutoff
 * sphere of that node, i.e. | |node - r_j| - cutoff | < margin.  The vertex score jumps by f(cutoff^-) (about
 * -0.004 per atom, reading S3) there, so an implementation in another precision may legitimately count that atom
 * on the other side; the parity tests exempt these nodes and assert that they are few.  Returns the number flagged. */
int64_t orc_grid_cutoff_flags(int np, const double *pxyz, const int dims[3], const double origin[3], double h,
                              double cutoff, double margin, uint8_t *flags)
{
    const int nx = dims[0], ny = dims[1], nz = dims[2];
    const int64_t nodes = (int64_t)nx * ny * nz;
    int64_t count = 0;
#pragma omp parallel for schedule(dynamic, 64) reduction(+ : count)
    for (int64_t m = 0; m < nodes; ++m) {
        int ix = (int)(m % nx), iy = (int)((m / nx) % ny), iz = (int)(m / ((int64_t)nx * ny));
        double mx = origin[0] + h * ix, my = origin[1] + h * iy, mz = origin[2] + h * iz;
        int near = 0;
        for (int j = 0; j < np && !near; ++j) {
            double dx = mx - pxyz[3 * j], dy = my - pxyz[3 * j + 1], dz = mz - pxyz[3 * j + 2];
            if (fabs(sqrt(dx * dx + dy * dy + dz * dz) - cutoff) < margin) near = 1;
        }
        flags[m] = (uint8_t)near;
        count += near;
    }
    return count;
}

/* NEXT-2 / eq. 4: per-vertex gradient of the vertex score, by the same brute force as O2. */
void orc_build_grid_grad(const orc_params *p, int np, const double *pxyz, const int32_t *ptype,
                         const int dims[3], const double origin[3], double h,
                         int n_lig_types, const int32_t *lig_types, double *GD)
{
    const int nx = dims[0], ny = dims[1], nz = dims[2];
    const int64_t nodes = (int64_t)nx * ny * nz;
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t m = 0; m < nodes; ++m) {
        int ix = (int)(m % nx), iy = (int)((m / nx) % ny), iz = (int)(m / ((int64_t)nx * ny));
        double mx = origin[0] + h * ix, my = origin[1] + h * iy, mz = origin[2] + h * iz;
        for (int t = 0; t < n_lig_types; ++t)
            for (int c = 0; c < 3; ++c) GD[((int64_t)t * 3 + c) * nodes + m] = 0.0;
        for (int j = 0; j < np; ++j) {
            double d[3] = {mx - pxyz[3 * j], my - pxyz[3 * j + 1], mz - pxyz[3 * j + 2]};
            double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
            if (!(r < p->cutoff) || r <= 0.0) continue;
            for (int t = 0; t < n_lig_types; ++t) {
                double dfdr;
                orc_pair(p, lig_types[t], ptype[j], r, &dfdr);
                for (int c = 0; c < 3; ++c) GD[((int64_t)t * 3 + c) * nodes + m] += dfdr * d[c] / r;
            }
        }
    }
}

/* ---------------------------------------------------------------------------------------
 * small vector / quaternion helpers
 * ------------------------------------------------------------------------------------- */
static void cross(const double a[3], const double b[3], double c[3])
{
    c[0] = a[1] * b[2] - a[2] * b[1];
    c[1] = a[2] * b[0] - a[0] * b[2];
    c[2] = a[0] * b[1] - a[1] * b[0];
}
static double dot(const double a[3], const double b[3]) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }

static void quat_normalize(double q[4])
{
    double n = sqrt(q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + q[3] * q[3]);
    if (n > 0.0) { q[0] /= n; q[1] /= n; q[2] /= n; q[3] /= n; }
    else { q[0] = 1.0; q[1] = q[2] = q[3] = 0.0; }
}
/* Hamilton product a*b, (w,x,y,z) */
static void quat_mul(const double a[4], const double b[4], double c[4])
{
    c[0] = a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3];
    c[1] = a[0] * b[1] + a[1] * b[0] + a[2] * b[3] - a[3] * b[2];
    c[2] = a[0] * b[2] - a[1] * b[3] + a[2] * b[0] + a[3] * b[1];
    c[3] = a[0] * b[3] + a[1] * b[2] - a[2] * b[1] + a[3] * b[0];
}
static void quat_from_rotvec(const double w[3], double q[4])
{
    double phi = sqrt(dot(w, w));
    if (phi < 1e-12) {
        q[0] = 1.0; q[1] = 0.5 * w[0]; q[2] = 0.5 * w[1]; q[3] = 0.5 * w[2];
    } else {
        double s = sin(0.5 * phi) / phi;
        q[0] = cos(0.5 * phi); q[1] = s * w[0]; q[2] = s * w[1]; q[3] = s * w[2];
    }
    quat_normalize(q);
}
static void quat_to_matrix(const double qin[4], double R[9])
{
    double q[4] = {qin[0], qin[1], qin[2], qin[3]};
    quat_normalize(q);
    double w = q[0], x = q[1], y = q[2], z = q[3];
    R[0] = 1 - 2 * (y * y + z * z); R[1] = 2 * (x * y - w * z);     R[2] = 2 * (x * z + w * y);
    R[3] = 2 * (x * y + w * z);     R[4] = 1 - 2 * (x * x + z * z); R[5] = 2 * (y * z - w * x);
    R[6] = 2 * (x * z - w * y);     R[7] = 2 * (y * z + w * x);     R[8] = 1 - 2 * (x * x + y * y);
}
/* rotate v about unit axis u by angle th (right-handed), Rodrigues */
static void rot_axis(const double u[3], double th, const double v[3], double out[3])
{
    double c = cos(th), s = sin(th), uxv[3];
    cross(u, v, uxv);
    double ud = dot(u, v);
    for (int k = 0; k < 3; ++k) out[k] = v[k] * c + uxv[k] * s + u[k] * ud * (1.0 - c);
}

void orc_pose_add(int T, const double *pose, const double *s, double *out)
{
    double qw[4], q[4];
    for (int k = 0; k < 3; ++k) out[k] = pose[k] + s[k];
    quat_from_rotvec(s + 3, qw);
    quat_mul(qw, pose + 3, q);
    quat_normalize(q);
    for (int k = 0; k < 4; ++k) out[3 + k] = q[k];
    for (int k = 0; k < T; ++k) out[7 + k] = pose[7 + k] + s[6 + k];
}

/* ---------------------------------------------------------------------------------------
 * O3 kinematics (reading S11).  pivot c = mean of the root-fragment reference atoms.
 * Fragment transforms parents-first: A_0 = id; A_{k+1}(y) = A_parent( Rot(u_k, theta_k)(y - ref[b_k]) + ref[b_k] ),
 * u_k = unit(ref[b_k] - ref[a_k]).  y_i = A_{frag(i)}(ref_i);  x_i = t + R(q)(y_i - c).
 * A_f is stored as y -> M_f y + v_f.
 * ------------------------------------------------------------------------------------- */
static void root_pivot(const orc_ligand *L, double c[3])
{
    int n = 0;
    c[0] = c[1] = c[2] = 0.0;
    for (int i = 0; i < L->N; ++i)
        if (L->frag[i] == 0) { c[0] += L->ref[3 * i]; c[1] += L->ref[3 * i + 1]; c[2] += L->ref[3 * i + 2]; ++n; }
    c[0] /= n; c[1] /= n; c[2] /= n;
}

void orc_coords(const orc_ligand *L, const double *pose, double *x)
{
    const int T = L->T;
    double *M = (double *)malloc(sizeof(double) * 9 * (T + 1));
    double *v = (double *)malloc(sizeof(double) * 3 * (T + 1));
    for (int k = 0; k < 9; ++k) M[k] = (k % 4 == 0) ? 1.0 : 0.0;
    v[0] = v[1] = v[2] = 0.0;
    for (int k = 0; k < T; ++k) {
        const double *pa = L->ref + 3 * L->tors_a[k], *pb = L->ref + 3 * L->tors_b[k];
        double u[3] = {pb[0] - pa[0], pb[1] - pa[1], pb[2] - pa[2]};
        double n = sqrt(dot(u, u));
        u[0] /= n; u[1] /= n; u[2] /= n;
        /* local map: y -> Rk (y - pb) + pb  =  Rk y + (pb - Rk pb) */
        double Rk[9], e[3], col[3];
        for (int c = 0; c < 3; ++c) {
            e[0] = e[1] = e[2] = 0.0; e[c] = 1.0;
            rot_axis(u, pose[7 + k], e, col);
            Rk[0 + c] = col[0]; Rk[3 + c] = col[1]; Rk[6 + c] = col[2];
        }
        double Rpb[3] = {Rk[0] * pb[0] + Rk[1] * pb[1] + Rk[2] * pb[2],
                         Rk[3] * pb[0] + Rk[4] * pb[1] + Rk[5] * pb[2],
                         Rk[6] * pb[0] + Rk[7] * pb[1] + Rk[8] * pb[2]};
        double lk[3] = {pb[0] - Rpb[0], pb[1] - Rpb[1], pb[2] - Rpb[2]};
        const double *Mp = M + 9 * L->tors_parent[k], *vp = v + 3 * L->tors_parent[k];
        double *Mc = M + 9 * (k + 1), *vc = v + 3 * (k + 1);
        for (int r = 0; r < 3; ++r) {
            for (int c = 0; c < 3; ++c)
                Mc[3 * r + c] = Mp[3 * r] * Rk[c] + Mp[3 * r + 1] * Rk[3 + c] + Mp[3 * r + 2] * Rk[6 + c];
            vc[r] = Mp[3 * r] * lk[0] + Mp[3 * r + 1] * lk[1] + Mp[3 * r + 2] * lk[2] + vp[r];
        }
    }
    double R[9], c[3];
    quat_to_matrix(pose + 3, R);
    root_pivot(L, c);
    for (int i = 0; i < L->N; ++i) {
        const double *Mf = M + 9 * L->frag[i], *vf = v + 3 * L->frag[i], *r0 = L->ref + 3 * i;
        double y[3];
        for (int r = 0; r < 3; ++r) y[r] = Mf[3 * r] * r0[0] + Mf[3 * r + 1] * r0[1] + Mf[3 * r + 2] * r0[2] + vf[r] - c[r];
        for (int r = 0; r < 3; ++r) x[3 * i + r] = pose[r] + R[3 * r] * y[0] + R[3 * r + 1] * y[1] + R[3 * r + 2] * y[2];
    }
    free(M);
    free(v);
}

/* ---------------------------------------------------------------------------------------
 * O4 inter term for one atom: trilinear energy (eq. 2), its partial
 * derivatives (eq. 3), clamp + quadratic wall (reading S7),
 * cell choice i0 = min(floor(u), n-2) (reading S8).
 * ------------------------------------------------------------------------------------- */
static void atom_inter(const orc_params *p, const orc_grid *g, int map, const double x[3],
                       double *e_grid, double *e_wall, double grad[3], double *face_margin, int *outside)
{
    int i0[3], clamped[3];
    double pf[3], over[3];
    const double h = g->h;
    *outside = 0;
    for (int c = 0; c < 3; ++c) {
        const int n = g->dims[c];
        double u = (x[c] - g->origin[c]) / h;
        over[c] = 0.0;
        clamped[c] = 0;
        if (u < 0.0) { over[c] = x[c] - g->origin[c]; u = 0.0; clamped[c] = 1; }
        else if (u > (double)(n - 1)) { over[c] = x[c] - (g->origin[c] + h * (n - 1)); u = (double)(n - 1); clamped[c] = 1; }
        int fl = (int)floor(u);
        i0[c] = fl < n - 2 ? fl : n - 2;
        pf[c] = u - (double)i0[c];
        if (clamped[c]) *outside = 1;
        if (face_margin) {
            double m = clamped[c] ? fabs(over[c]) : fmin(pf[c], 1.0 - pf[c]) * h;
            if (m < *face_margin) *face_margin = m;
        }
    }
    const int nx = g->dims[0], ny = g->dims[1], nz = g->dims[2];
    const double *G = g->data + (int64_t)map * nx * ny * nz;
    double e = 0.0, gx = 0.0, gy = 0.0, gz = 0.0;
    for (int l = 0; l <= 1; ++l)
        for (int m = 0; m <= 1; ++m)
            for (int n = 0; n <= 1; ++n) {
                double wx = l ? pf[0] : 1.0 - pf[0];
                double wy = m ? pf[1] : 1.0 - pf[1];
                double wz = n ? pf[2] : 1.0 - pf[2];
                double val = G[((int64_t)(i0[2] + n) * ny + (i0[1] + m)) * nx + (i0[0] + l)];
                e += wx * wy * wz * val;                       /* eq. 2 */
                gx += (2 * l - 1) / h * wy * wz * val;         /* eq. 3, x component */
                gy += wx * (2 * m - 1) / h * wz * val;         /* eq. 3, y component */
                gz += wx * wy * (2 * n - 1) / h * val;         /* eq. 3, z component */
            }
    if (g->gdata) {                                            /* eq. 4: the vertex gradients, interpolated with eq. 2's weights */
        const int64_t nodes = (int64_t)nx * ny * nz;
        const double *GD = g->gdata + (int64_t)map * 3 * nodes;
        gx = gy = gz = 0.0;
        for (int l = 0; l <= 1; ++l)
            for (int m = 0; m <= 1; ++m)
                for (int n = 0; n <= 1; ++n) {
                    double w = (l ? pf[0] : 1.0 - pf[0]) * (m ? pf[1] : 1.0 - pf[1]) * (n ? pf[2] : 1.0 - pf[2]);
                    int64_t node = ((int64_t)(i0[2] + n) * ny + (i0[1] + m)) * nx + (i0[0] + l);
                    gx += w * GD[node];
                    gy += w * GD[nodes + node];
                    gz += w * GD[2 * nodes + node];
                }
    }
    double ew = 0.0;
    double gg[3] = {gx, gy, gz};
    for (int c = 0; c < 3; ++c) {
        if (clamped[c]) gg[c] = 0.0;                           /* lookup is constant along a clamped axis */
        ew += p->k_wall * over[c] * over[c];
        gg[c] += 2.0 * p->k_wall * over[c];
        grad[c] = gg[c];
    }
    *e_grid = e;
    *e_wall = ew;
}

/* ---------------------------------------------------------------------------------------
 * O4-O7: total E = E_grid + E_wall + E_intra and its gradient wrt (t, rotation about t, theta).
 * ------------------------------------------------------------------------------------- */
double orc_eval(const orc_params *p, const orc_grid *g, const orc_ligand *L,
                const double *pose, double terms[3], double *grad, orc_diag *diag)
{
    const int N = L->N, T = L->T;
    double *x = (double *)malloc(sizeof(double) * 3 * N);
    double *gx = (double *)calloc(3 * N, sizeof(double));
    double e_grid = 0.0, e_wall = 0.0, e_intra = 0.0;
    double face_margin = 1e300, kink_margin = 1e300, cutoff_margin = 1e300;
    int n_in = 0, n_out = 0;
    orc_coords(L, pose, x);
    for (int i = 0; i < N; ++i) {
        double eg, ew, ga[3];
        int outside;
        int map = g->type_to_map[L->type[i]];
        atom_inter(p, g, map, x + 3 * i, &eg, &ew, ga, diag ? &face_margin : NULL, &outside);
        e_grid += eg;
        e_wall += ew;
        n_out += outside;
        for (int c = 0; c < 3; ++c) gx[3 * i + c] += ga[c];
    }
    /* O5 intra-ligand pairs */
    for (int k = 0; k < L->P; ++k) {
        int i = L->pairs[2 * k], j = L->pairs[2 * k + 1];
        double d[3] = {x[3 * i] - x[3 * j], x[3 * i + 1] - x[3 * j + 1], x[3 * i + 2] - x[3 * j + 2]};
        double r = sqrt(dot(d, d)), dfdr;
        e_intra += orc_pair(p, L->type[i], L->type[j], r, &dfdr);
        if (r < p->cutoff) ++n_in;
        if (diag) {
            kink_margin = fmin(kink_margin, pair_kink_margin(p, L->type[i], L->type[j], r));
            cutoff_margin = fmin(cutoff_margin, fabs(r - p->cutoff));
        }
        if (r > 1e-12)
            for (int c = 0; c < 3; ++c) {
                gx[3 * i + c] += dfdr * d[c] / r;
                gx[3 * j + c] -= dfdr * d[c] / r;
            }
    }
    if (terms) { terms[0] = e_grid; terms[1] = e_wall; terms[2] = e_intra; }
    if (grad) {
        /* O6 chain rule */
        for (int k = 0; k < 6 + T; ++k) grad[k] = 0.0;
        for (int i = 0; i < N; ++i) {
            double lever[3] = {x[3 * i] - pose[0], x[3 * i + 1] - pose[1], x[3 * i + 2] - pose[2]}, tq[3];
            cross(lever, gx + 3 * i, tq);
            for (int c = 0; c < 3; ++c) { grad[c] += gx[3 * i + c]; grad[3 + c] += tq[c]; }
        }
        for (int k = 0; k < T; ++k) {
            /* subtree(k) = fragment k+1 and every fragment whose parent chain passes through it */
            const double *xa = x + 3 * L->tors_a[k], *xb = x + 3 * L->tors_b[k];
            double u[3] = {xb[0] - xa[0], xb[1] - xa[1], xb[2] - xa[2]};
            double n = sqrt(dot(u, u));
            u[0] /= n; u[1] /= n; u[2] /= n;
            double acc[3] = {0, 0, 0};
            for (int i = 0; i < N; ++i) {
                int f = L->frag[i], in_sub = 0;
                while (f > 0) {
                    if (f == k + 1) { in_sub = 1; break; }
                    f = L->tors_parent[f - 1];
                }
                if (!in_sub) continue;
                double lever[3] = {x[3 * i] - xb[0], x[3 * i + 1] - xb[1], x[3 * i + 2] - xb[2]}, tq[3];
                cross(lever, gx + 3 * i, tq);
                acc[0] += tq[0]; acc[1] += tq[1]; acc[2] += tq[2];
            }
            grad[6 + k] = dot(u, acc);
        }
    }
    if (diag) {
        diag->face_margin = face_margin;
        diag->kink_margin = kink_margin;
        diag->cutoff_margin = cutoff_margin;
        diag->pairs_in_range = n_in;
        diag->atoms_outside = n_out;
    }
    free(x);
    free(gx);
    return e_grid + e_wall + e_intra;   /* O7 */
}

void orc_score_batch(const orc_params *p, const orc_grid *g, const orc_ligand *L, int64_t n,
                     const double *poses, double *E, double *grad, double *terms, orc_diag *diag)
{
    const int T = L->T;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t k = 0; k < n; ++k) {
        double tr[3];
        E[k] = orc_eval(p, g, L, poses + k * (7 + T), tr, grad ? grad + k * (6 + T) : NULL, diag ? diag + k : NULL);
        if (terms) { terms[3 * k] = tr[0]; terms[3 * k + 1] = tr[1]; terms[3 * k + 2] = tr[2]; }
    }
}

/* ---------------------------------------------------------------------------------------
 * Diagnostic only (changes no result): the conditioning scale of every gradient component,
 * A_k = sum over atoms of the ABSOLUTE values of the terms that orc_eval adds up for grad[k]
 * (per-atom force taken as |grid gradient| + sum over pairs |pair force|).  A working precision
 * eps can resolve grad[k] only to ~eps * A_k; the parity tests use A_k to tell a wrong gradient
 * from a cancellation the fp32 kernel cannot resolve (reading S20').
 * ------------------------------------------------------------------------------------- */
void orc_grad_cond(const orc_params *p, const orc_grid *g, const orc_ligand *L, const double *pose, double *A)
{
    const int N = L->N, T = L->T;
    double *x = (double *)malloc(sizeof(double) * 3 * N);
    double *ax = (double *)calloc(3 * N, sizeof(double));
    orc_coords(L, pose, x);
    for (int i = 0; i < N; ++i) {
        double eg, ew, ga[3];
        int outside;
        atom_inter(p, g, g->type_to_map[L->type[i]], x + 3 * i, &eg, &ew, ga, NULL, &outside);
        for (int c = 0; c < 3; ++c) ax[3 * i + c] += fabs(ga[c]);
    }
    for (int k = 0; k < L->P; ++k) {
        int i = L->pairs[2 * k], j = L->pairs[2 * k + 1];
        double d[3] = {x[3 * i] - x[3 * j], x[3 * i + 1] - x[3 * j + 1], x[3 * i + 2] - x[3 * j + 2]};
        double r = sqrt(dot(d, d)), dfdr;
        orc_pair(p, L->type[i], L->type[j], r, &dfdr);
        if (r > 1e-12)
            for (int c = 0; c < 3; ++c) {
                ax[3 * i + c] += fabs(dfdr * d[c] / r);
                ax[3 * j + c] += fabs(dfdr * d[c] / r);
            }
    }
    for (int k = 0; k < 6 + T; ++k) A[k] = 0.0;
    for (int i = 0; i < N; ++i) {
        const double *a = ax + 3 * i;
        double l[3] = {fabs(x[3 * i] - pose[0]), fabs(x[3 * i + 1] - pose[1]), fabs(x[3 * i + 2] - pose[2])};
        for (int c = 0; c < 3; ++c) A[c] += a[c];
        A[3] += l[1] * a[2] + l[2] * a[1];
        A[4] += l[2] * a[0] + l[0] * a[2];
        A[5] += l[0] * a[1] + l[1] * a[0];
    }
    for (int k = 0; k < T; ++k) {
        const double *xa = x + 3 * L->tors_a[k], *xb = x + 3 * L->tors_b[k];
        double u[3] = {xb[0] - xa[0], xb[1] - xa[1], xb[2] - xa[2]};
        double n = sqrt(dot(u, u));
        for (int i = 0; i < N; ++i) {
            int f = L->frag[i], in_sub = 0;
            while (f > 0) {
                if (f == k + 1) { in_sub = 1; break; }
                f = L->tors_parent[f - 1];
            }
            if (!in_sub) continue;
            const double *a = ax + 3 * i;
            double l[3] = {fabs(x[3 * i] - xb[0]), fabs(x[3 * i + 1] - xb[1]), fabs(x[3 * i + 2] - xb[2])};
            A[6 + k] += (fabs(u[0]) * (l[1] * a[2] + l[2] * a[1]) + fabs(u[1]) * (l[2] * a[0] + l[0] * a[2]) +
                         fabs(u[2]) * (l[0] * a[1] + l[1] * a[0])) / n;
        }
    }
    free(x);
    free(ax);
}

void orc_grad_cond_batch(const orc_params *p, const orc_grid *g, const orc_ligand *L, int64_t n,
                         const double *poses, double *A)
{
    const int T = L->T;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t k = 0; k < n; ++k) orc_grad_cond(p, g, L, poses + k * (7 + T), A + k * (6 + T));
}

/* ---------------------------------------------------------------------------------------
 * O8 BFGS with backtracking (Nocedal-Wright inverse update).
 * Every constant is a reading (S12) and a field of orc_params.
 *
 * The optimizer is generic over the objective (`fn` returns f and writes the gradient) and
 * over the retraction x (+) s (`add`), so that the pin tests can run it on closed-form
 * quadratics; orc_local_opt instantiates it with the docking objective and orc_pose_add.
 * `obs` (nullable) is called after every accepted iteration with (it, f, H, s, y, updated).
 *
 * One iteration is written once (bfgs_iteration) and used by the full loop (orc_bfgs) and by the
 * single-step replay of the iteration-level teacher-forced parity test (orc_bfgs_step).
 * ------------------------------------------------------------------------------------- */
typedef struct {
    int n, np_;
    double *H, *A, *B, *x, *xt, *gr, *gt, *d, *s, *y;
    double f;
    int fresh;        /* H is still the identity (no update applied since the start or the last reset) */
    int ne;           /* evaluations so far */
} bfgs_state;

static void bfgs_alloc(bfgs_state *S, int n, int np_)
{
    S->n = n; S->np_ = np_;
    S->H = (double *)malloc(sizeof(double) * n * n);
    S->A = (double *)malloc(sizeof(double) * n * n);
    S->B = (double *)malloc(sizeof(double) * n * n);
    S->x = (double *)malloc(sizeof(double) * np_); S->xt = (double *)malloc(sizeof(double) * np_);
    S->gr = (double *)malloc(sizeof(double) * n); S->gt = (double *)malloc(sizeof(double) * n);
    S->d = (double *)malloc(sizeof(double) * n); S->s = (double *)malloc(sizeof(double) * n); S->y = (double *)malloc(sizeof(double) * n);
    S->f = 0.0; S->fresh = 1; S->ne = 0;
}
static void bfgs_free(bfgs_state *S)
{
    free(S->H); free(S->A); free(S->B); free(S->x); free(S->xt); free(S->gr); free(S->gt); free(S->d); free(S->s); free(S->y);
}

/* One iteration from the state (x, f, gr, H, fresh).  Returns 0 if a step was accepted (state advanced),
 * ORC_EXIT_GTOL if ||g|| < gtol (nothing done), ORC_EXIT_LINESEARCH if no trial was acceptable (state unchanged).
 * `rec` (nullable) receives the decision scalars of the iteration. */
static int bfgs_iteration(const orc_params *p, bfgs_state *S, orc_objective_fn fn, orc_retract_fn add, void *ctx,
                          orc_iter_rec *rec)
{
    const int n = S->n, np_ = S->np_;
    double *H = S->H, *A = S->A, *B = S->B, *x = S->x, *xt = S->xt, *gr = S->gr, *gt = S->gt, *d = S->d, *s = S->s, *y = S->y;
    if (rec) { memset(rec, 0, sizeof(*rec)); rec->f = S->f; rec->fresh_in = S->fresh; }
    double gn = 0.0;
    for (int k = 0; k < n; ++k) gn += gr[k] * gr[k];
    if (rec) rec->gnorm = sqrt(gn);
    if (sqrt(gn) < p->bfgs_gtol) { if (rec) rec->status = ORC_EXIT_GTOL; return ORC_EXIT_GTOL; }
    double gp = 0.0;
    for (int r = 0; r < n; ++r) {                      /* d = -H g */
        double a = 0.0;
        for (int c = 0; c < n; ++c) a += H[r * n + c] * gr[c];
        d[r] = -a;
        gp += gr[r] * d[r];
    }
    if (gp >= 0.0) {                                   /* not a descent direction: reset H = I */
        for (int r = 0; r < n; ++r) for (int c = 0; c < n; ++c) H[r * n + c] = (r == c) ? 1.0 : 0.0;
        S->fresh = 1;
        gp = 0.0;
        for (int r = 0; r < n; ++r) { d[r] = -gr[r]; gp += gr[r] * d[r]; }
        if (rec) rec->reset = 1;
    }
    double alpha = 1.0;
    if (S->fresh) {                                    /* alpha0 = min(1, 1/||d||) while H = I */
        double dn = 0.0;
        for (int k = 0; k < n; ++k) dn += d[k] * d[k];
        dn = sqrt(dn);
        if (dn > 1.0) alpha = 1.0 / dn;
    }
    if (rec) { rec->gp = gp; rec->alpha0 = alpha; }
    int ok = 0;
    double ft = S->f;
    for (int trial = 0; trial < p->bfgs_max_trials; ++trial) {
        for (int k = 0; k < n; ++k) s[k] = alpha * d[k];
        add(ctx, x, s, xt);
        ft = fn(ctx, xt, gt);
        ++S->ne;
        if (rec) {
            rec->trials = trial + 1;
            rec->alpha = alpha;
            if (trial < ORC_MAX_TRIALS) rec->armijo_margin[trial] = (ft - S->f) - p->bfgs_c1 * alpha * gp;
        }
        if (ft - S->f <= p->bfgs_c1 * alpha * gp) { ok = 1; break; }   /* Armijo */
        alpha *= p->bfgs_shrink;
    }
    if (!ok) { if (rec) rec->status = ORC_EXIT_LINESEARCH; return ORC_EXIT_LINESEARCH; }
    double ys = 0.0, yy = 0.0, ss = 0.0;
    for (int k = 0; k < n; ++k) {
        y[k] = gt[k] - gr[k];
        ys += y[k] * s[k]; yy += y[k] * y[k]; ss += s[k] * s[k];
    }
    memcpy(x, xt, sizeof(double) * np_);
    memcpy(gr, gt, sizeof(double) * n);
    S->f = ft;
    int updated = 0;
    if (rec) { rec->f_new = ft; rec->curv_margin = ys - p->bfgs_curv_eps * sqrt(ss) * sqrt(yy); }
    if (ys > p->bfgs_curv_eps * sqrt(ss) * sqrt(yy)) {
        if (S->fresh) {                                /* first update: H = (y.s / y.y) I */
            double sc = ys / yy;
            for (int r = 0; r < n; ++r) for (int c = 0; c < n; ++c) H[r * n + c] = (r == c) ? sc : 0.0;
            S->fresh = 0;
        }
        /* H <- (I - rho s y^T) H (I - rho y s^T) + rho s s^T */
        double rho = 1.0 / ys;
        for (int r = 0; r < n; ++r) for (int c = 0; c < n; ++c) {   /* A = (I - rho s y^T) H */
            double a = H[r * n + c];
            for (int k = 0; k < n; ++k) a -= rho * s[r] * y[k] * H[k * n + c];
            A[r * n + c] = a;
        }
        for (int r = 0; r < n; ++r) for (int c = 0; c < n; ++c) {   /* B = A (I - rho y s^T) + rho s s^T */
            double a = A[r * n + c];
            for (int k = 0; k < n; ++k) a -= A[r * n + k] * rho * y[k] * s[c];
            B[r * n + c] = a + rho * s[r] * s[c];
        }
        memcpy(H, B, sizeof(double) * n * n);
        updated = 1;
    }
    if (rec) { rec->updated = updated; rec->fresh_out = S->fresh; }
    return 0;
}

double orc_bfgs(const orc_params *p, int n, int np_, int cap, const double *x0,
                orc_objective_fn fn, orc_retract_fn add, void *ctx,
                double *x_out, int *iters, int *evals, orc_observer_fn obs, void *obs_ctx,
                int *exit_reason, orc_iter_rec *recs, int max_recs)
{
    bfgs_state S;
    bfgs_alloc(&S, n, np_);
    int it = 0, why = ORC_EXIT_CAP;
    memcpy(S.x, x0, sizeof(double) * np_);
    S.f = fn(ctx, S.x, S.gr);
    ++S.ne;
    for (int r = 0; r < n; ++r) for (int c = 0; c < n; ++c) S.H[r * n + c] = (r == c) ? 1.0 : 0.0;
    for (it = 0; it < cap; ++it) {
        orc_iter_rec tmp;
        const int st = bfgs_iteration(p, &S, fn, add, ctx, (recs && it < max_recs) ? &recs[it] : &tmp);
        if (st != 0) { why = st; break; }
        if (obs) obs(obs_ctx, it, S.f, S.H, S.s, S.y, (recs && it < max_recs) ? recs[it].updated : tmp.updated);
    }
    memcpy(x_out, S.x, sizeof(double) * np_);
    if (iters) *iters = it;
    if (evals) *evals = S.ne;
    if (exit_reason) *exit_reason = why;
    const double f = S.f;
    bfgs_free(&S);
    return f;
}

typedef struct {
    const orc_params *p; const orc_grid *g; const orc_ligand *L;
    double *min_cutoff_margin;   /* diagnostic, nullable: min over all evaluations of orc_diag.cutoff_margin */
} dock_ctx;

/* Diagnostic switch for the "chaos ceiling" measurement; OFF by default and never
 * switched on by anything but tests/parity.py: when on, the docking objective handed to the optimizers returns the
 * oracle's energy and gradient rounded to a (24 - drop_bits)-bit significand: drop_bits = 0 is fp32 correctly
 * rounded -- the best any single-precision evaluator could do --, drop_bits = 3 an fp32 result that is off by up to
 * 4 ulp, which is what a sum of a few hundred fp32 terms delivers.  Comparing the oracle with itself under this
 * switch says how far a free-running local optimisation / search may legitimately drift for a reason that is not an
 * implementation difference.  drop_bits < 0 switches it off. */
static int g_eval_drop_bits = -1;
void orc_diag_round_eval_fp32(int drop_bits) { g_eval_drop_bits = drop_bits; }
static double round_sig(double x, int bits)
{
    if (x == 0.0 || !isfinite(x)) return x;
    int e;
    double m = frexp(x, &e);                       /* x = m 2^e, 0.5 <= |m| < 1 */
    return ldexp(nearbyint(ldexp(m, bits)), e - bits);
}

/* ---------------------------------------------------------------------------------------
 * O8' Barzilai-Borwein ("BB only needs a vector inner product to estimate the step
 * length and does not need to perform line search"; ref. 37).  Reading S13:
 *   alpha_0 = bb_step / |g_0|;  alpha_k = s.s / s.y  (s = x_k - x_{k-1} in tangent coordinates,
 *   y = g_k - g_{k-1}) if s.y > curv_eps |s| |y|, else bb_fallback / |g_k|;  alpha_k |g_k| <= bb_step.
 * ------------------------------------------------------------------------------------- */
/* One iteration from the state (x, f, gr) and the previous step (s, y; unused when `first`).  Returns 0 if the step was
 * taken (state advanced: x, f, gr, s, y), ORC_EXIT_GTOL if ||g|| < gtol (nothing done).  Written once, used by the
 * full loop (orc_bb) and by the single-step replay of the iteration-level parity test (orc_bb_step). */
static int bb_iteration(const orc_params *p, int n, int np_, orc_objective_fn fn, orc_retract_fn add, void *ctx,
                        int first, double *x, double *f, double *gr, double *s, double *y, double *xn, double *gn,
                        int *ne, orc_bb_rec *rec)
{
    if (rec) { memset(rec, 0, sizeof(*rec)); rec->f = *f; }
    double g2 = 0.0;
    for (int k = 0; k < n; ++k) g2 += gr[k] * gr[k];
    const double gnorm = sqrt(g2);
    if (rec) rec->gnorm = gnorm;
    if (gnorm < p->bfgs_gtol) { if (rec) rec->status = ORC_EXIT_GTOL; return ORC_EXIT_GTOL; }
    double alpha;
    if (first) alpha = p->bb_step / gnorm;
    else {
        double sy = 0.0, ss = 0.0, yy = 0.0;
        for (int k = 0; k < n; ++k) { sy += s[k] * y[k]; ss += s[k] * s[k]; yy += y[k] * y[k]; }
        alpha = (sy > p->bfgs_curv_eps * sqrt(ss) * sqrt(yy)) ? ss / sy : p->bb_fallback / gnorm;
        if (rec) { rec->branch = (sy > p->bfgs_curv_eps * sqrt(ss) * sqrt(yy)) ? 1 : 2; rec->sy_margin = sy - p->bfgs_curv_eps * sqrt(ss) * sqrt(yy); }
    }
    if (rec) rec->cap_margin = alpha * gnorm - p->bb_step;
    if (alpha * gnorm > p->bb_step) { alpha = p->bb_step / gnorm; if (rec) rec->capped = 1; }
    for (int k = 0; k < n; ++k) s[k] = -alpha * gr[k];
    add(ctx, x, s, xn);
    const double fnew = fn(ctx, xn, gn);
    ++*ne;
    for (int k = 0; k < n; ++k) { y[k] = gn[k] - gr[k]; gr[k] = gn[k]; }
    memcpy(x, xn, sizeof(double) * np_);
    *f = fnew;
    if (rec) { rec->alpha = alpha; rec->f_new = fnew; }
    return 0;
}

double orc_bb(const orc_params *p, int n, int np_, int cap, const double *x0,
              orc_objective_fn fn, orc_retract_fn add, void *ctx,
              double *x_out, int *iters, int *evals, orc_observer_fn obs, void *obs_ctx, int *exit_reason)
{
    int why = ORC_EXIT_CAP;
    double *x = (double *)malloc(sizeof(double) * np_), *xn = (double *)malloc(sizeof(double) * np_);
    double *gr = (double *)malloc(sizeof(double) * n), *gn = (double *)malloc(sizeof(double) * n);
    double *s = (double *)malloc(sizeof(double) * n), *y = (double *)malloc(sizeof(double) * n);
    int it = 0, ne = 0;
    memcpy(x, x0, sizeof(double) * np_);
    double f = fn(ctx, x, gr);
    ++ne;
    double fbest = f;
    memcpy(x_out, x, sizeof(double) * np_);
    for (it = 0; it < cap; ++it) {
        if (bb_iteration(p, n, np_, fn, add, ctx, it == 0, x, &f, gr, s, y, xn, gn, &ne, NULL) != 0) { why = ORC_EXIT_GTOL; break; }
        if (obs) obs(obs_ctx, it, f, NULL, s, y, 1);
        if (f < fbest) { fbest = f; memcpy(x_out, x, sizeof(double) * np_); }
    }
    if (iters) *iters = it;
    if (evals) *evals = ne;
    if (exit_reason) *exit_reason = why;
    free(x); free(xn); free(gr); free(gn); free(s); free(y);
    return fbest;
}

static double dock_fn(void *c, const double *x, double *grad)
{
    dock_ctx *k = (dock_ctx *)c;
    orc_diag dg;
    double e = orc_eval(k->p, k->g, k->L, x, NULL, grad, k->min_cutoff_margin ? &dg : NULL);
    if (k->min_cutoff_margin && dg.cutoff_margin < *k->min_cutoff_margin) *k->min_cutoff_margin = dg.cutoff_margin;
    if (g_eval_drop_bits >= 0) {
        e = round_sig(e, 24 - g_eval_drop_bits);
        for (int i = 0; i < 6 + k->L->T; ++i) grad[i] = round_sig(grad[i], 24 - g_eval_drop_bits);
    }
    return e;
}
static void dock_add(void *c, const double *x, const double *s, double *out)
{
    orc_pose_add(((dock_ctx *)c)->L->T, x, s, out);
}

double orc_local_opt_ex(const orc_params *p, const orc_grid *g, const orc_ligand *L, int cap,
                        const double *pose_in, double *pose_out, int *iters, int *evals, int *exit_reason,
                        orc_iter_rec *recs, int max_recs)
{
    const int T = L->T;
    dock_ctx ctx = {p, g, L, NULL};
    double *x0 = (double *)malloc(sizeof(double) * (7 + T));
    memcpy(x0, pose_in, sizeof(double) * (7 + T));
    quat_normalize(x0 + 3);
    double f;
    if (p->optimizer == 1) f = orc_bb(p, 6 + T, 7 + T, cap, x0, dock_fn, dock_add, &ctx, pose_out, iters, evals, NULL, NULL, exit_reason);
    else f = orc_bfgs(p, 6 + T, 7 + T, cap, x0, dock_fn, dock_add, &ctx, pose_out, iters, evals, NULL, NULL, exit_reason, recs, max_recs);
    free(x0);
    return f;
}

double orc_local_opt(const orc_params *p, const orc_grid *g, const orc_ligand *L, int cap,
                     const double *pose_in, double *pose_out, int *iters, int *evals)
{
    return orc_local_opt_ex(p, g, L, cap, pose_in, pose_out, iters, evals, NULL, NULL, 0);
}

/* Diagnostic for the iteration-level teacher-forced parity test (SURVEY.md 8(c) parity protocol; DESIGN.md
 * "Parity levels"): ONE iteration of O8 on the docking objective from a GIVEN state -- pose x (quaternion used
 * as given), inverse Hessian H [n][n], the flag `fresh` (H is the identity of the start / of a reset) and,
 * optionally, the gradient g_in at x (NULL: evaluated here).  The energy at x and at every trial point is
 * evaluated here, in double.  Returns the status (0 = step accepted,
 * ORC_EXIT_GTOL, ORC_EXIT_LINESEARCH); x_new / H_new (nullable) receive the state after the iteration. */
int orc_bfgs_step(const orc_params *p, const orc_grid *g, const orc_ligand *L,
                  const double *x, const double *g_in, const double *H, int fresh, orc_iter_rec *rec, double *x_new, double *H_new)
{
    const int n = 6 + L->T, np_ = 7 + L->T;
    double mcm = 1e300;
    dock_ctx ctx = {p, g, L, &mcm};
    bfgs_state S;
    bfgs_alloc(&S, n, np_);
    memcpy(S.x, x, sizeof(double) * np_);
    memcpy(S.H, H, sizeof(double) * n * n);
    S.fresh = fresh;
    S.f = dock_fn(&ctx, S.x, S.gr);
    if (g_in) memcpy(S.gr, g_in, sizeof(double) * n);      /* the recorded gradient is part of the given state */
    const int st = bfgs_iteration(p, &S, dock_fn, dock_add, &ctx, rec);
    if (rec) rec->min_cutoff_margin = mcm;
    if (x_new) memcpy(x_new, S.x, sizeof(double) * np_);
    if (H_new) memcpy(H_new, S.H, sizeof(double) * n * n);
    bfgs_free(&S);
    return st;
}

void orc_bfgs_step_batch(const orc_params *p, const orc_grid *g, const orc_ligand *L, int64_t n_states,
                         const double *x, const double *g_in, const double *H, const int32_t *fresh,
                         orc_iter_rec *recs, double *x_new, double *H_new)
{
    const int n = 6 + L->T, np_ = 7 + L->T;
#pragma omp parallel for schedule(dynamic, 8)
    for (int64_t k = 0; k < n_states; ++k)
        orc_bfgs_step(p, g, L, x + k * np_, g_in ? g_in + k * n : NULL, H + k * n * n, fresh[k], recs + k,
                      x_new ? x_new + k * np_ : NULL, H_new ? H_new + k * n * n : NULL);
}

/* ONE O8' iteration on the docking objective from a GIVEN state: pose x, gradient g_in at x (NULL: evaluated here),
 * previous step s_prev / y_prev (tangent coordinates; ignored when `first`).  Energies are evaluated here, in double. */
int orc_bb_step(const orc_params *p, const orc_grid *g, const orc_ligand *L, const double *x, const double *g_in,
                const double *s_prev, const double *y_prev, int first, orc_bb_rec *rec, double *x_new)
{
    const int n = 6 + L->T, np_ = 7 + L->T;
    double mcm = 1e300;
    dock_ctx ctx = {p, g, L, &mcm};
    double *xx = (double *)malloc(sizeof(double) * np_), *xn = (double *)malloc(sizeof(double) * np_);
    double *gr = (double *)malloc(sizeof(double) * n), *gn = (double *)malloc(sizeof(double) * n);
    double *s = (double *)calloc(n, sizeof(double)), *y = (double *)calloc(n, sizeof(double));
    memcpy(xx, x, sizeof(double) * np_);
    double f = dock_fn(&ctx, xx, gr);
    if (g_in) memcpy(gr, g_in, sizeof(double) * n);
    if (!first) { memcpy(s, s_prev, sizeof(double) * n); memcpy(y, y_prev, sizeof(double) * n); }
    int ne = 0;
    const int st = bb_iteration(p, n, np_, dock_fn, dock_add, &ctx, first, xx, &f, gr, s, y, xn, gn, &ne, rec);
    if (rec) rec->min_cutoff_margin = mcm;
    if (x_new) memcpy(x_new, xx, sizeof(double) * np_);
    free(xx); free(xn); free(gr); free(gn); free(s); free(y);
    return st;
}

void orc_bb_step_batch(const orc_params *p, const orc_grid *g, const orc_ligand *L, int64_t n_states,
                       const double *x, const double *g_in, const double *s_prev, const double *y_prev,
                       const int32_t *first, orc_bb_rec *recs, double *x_new)
{
    const int n = 6 + L->T, np_ = 7 + L->T;
#pragma omp parallel for schedule(dynamic, 8)
    for (int64_t k = 0; k < n_states; ++k)
        orc_bb_step(p, g, L, x + k * np_, g_in ? g_in + k * n : NULL, s_prev + k * n, y_prev + k * n, first[k],
                    recs + k, x_new ? x_new + k * np_ : NULL);
}

/* batch of independent local optimisations (OpenMP over poses): poses [n][7+T] -> out_pose, out_e [n],
 * out_info [n][3] = (iters, evals, exit reason) */
void orc_local_opt_batch(const orc_params *p, const orc_grid *g, const orc_ligand *L, int cap, int64_t n,
                         const double *poses, double *out_pose, double *out_e, int32_t *out_info)
{
    const int np_ = 7 + L->T;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t k = 0; k < n; ++k) {
        int it, ne, why;
        out_e[k] = orc_local_opt_ex(p, g, L, cap, poses + k * np_, out_pose + k * np_, &it, &ne, &why, NULL, 0);
        out_info[3 * k] = it; out_info[3 * k + 1] = ne; out_info[3 * k + 2] = why;
    }
}

/* ---------------------------------------------------------------------------------------
 * O9 Monte Carlo (readings S14-S16; R-rules).
 * ------------------------------------------------------------------------------------- */
void orc_init_pose(const double box_center[3], const double box_size[3], int T,
                   uint64_t seed, uint32_t system, uint32_t copy, double *pose)
{
    uint32_t r[4];
    draw(seed, system, copy, 0xFFFFFFFFu, 0, r);
    for (int c = 0; c < 3; ++c) pose[c] = box_center[c] - 0.5 * box_size[c] + u24(r[c]) * box_size[c];
    draw(seed, system, copy, 0xFFFFFFFFu, 1, r);
    double u1 = u24(r[0]), u2 = u24(r[1]), u3 = u24(r[2]);
    pose[3] = sqrt(u1) * cos(2.0 * PI * u3);
    pose[4] = sqrt(1.0 - u1) * sin(2.0 * PI * u2);
    pose[5] = sqrt(1.0 - u1) * cos(2.0 * PI * u2);
    pose[6] = sqrt(u1) * sin(2.0 * PI * u3);
    for (int k = 0; k < T; ++k) {
        if (k % 4 == 0) draw(seed, system, copy, 0xFFFFFFFFu, 2 + (uint32_t)(k / 4), r);
        pose[7 + k] = PI * (2.0 * u24(r[k % 4]) - 1.0);
    }
    for (int k = 0; k < 7 + T; ++k) pose[k] = (double)(float)pose[k];   /* stored fp32 once (S16) */
}

/* NEXT-3 (Fig. 3): the search space is the intersection of the box with the union of balls of
 * radius `radius` centred at the predicted site points; "the initial ligand positions are not fully random but
 * restrained to the searching space".  Reading S22: rejection sampling of the translation -- attempt a = 0..255
 * draws t uniform in the box from Philox slot 0x100 + a (counter step 0xFFFFFFFF as in S16) and the first t
 * inside some ball is kept; if none is, t = site point (copy mod n_site).  Orientation and torsions as S16. */
void orc_init_pose_site(const double box_center[3], const double box_size[3], int T,
                        uint64_t seed, uint32_t system, uint32_t copy,
                        int n_site, const double *site_xyz, double radius, double *pose)
{
    orc_init_pose(box_center, box_size, T, seed, system, copy, pose);      /* q, theta (and a t that is replaced) */
    uint32_t r[4];
    int found = 0;
    double t[3];
    for (int a = 0; a < 256 && !found; ++a) {
        draw(seed, system, copy, 0xFFFFFFFFu, 0x100u + (uint32_t)a, r);
        for (int c = 0; c < 3; ++c) t[c] = box_center[c] - 0.5 * box_size[c] + u24(r[c]) * box_size[c];
        for (int k = 0; k < n_site && !found; ++k) {
            const double dx = t[0] - site_xyz[3 * k], dy = t[1] - site_xyz[3 * k + 1], dz = t[2] - site_xyz[3 * k + 2];
            if (dx * dx + dy * dy + dz * dz <= radius * radius) found = 1;
        }
    }
    if (!found)
        for (int c = 0; c < 3; ++c) t[c] = site_xyz[3 * (copy % (uint32_t)n_site) + c];
    for (int c = 0; c < 3; ++c) pose[c] = (double)(float)t[c];
}

int orc_mc_perturb(const orc_params *p, int T, uint64_t seed, uint32_t system, uint32_t copy,
                   uint32_t step, const double *pose, double *cand)
{
    uint32_t r[4];
    draw(seed, system, copy, step, 0, r);
    const uint32_t K = T > 0 ? 3u : 2u;
    int kind = (int)(((uint64_t)r[0] * K) >> 32);
    memcpy(cand, pose, sizeof(double) * (7 + T));
    if (kind == 0) {
        for (int c = 0; c < 3; ++c) cand[c] = pose[c] + p->amp_trans * (2.0 * u24(r[1 + c]) - 1.0);
    } else if (kind == 1) {
        double w[3], qw[4], q[4];
        for (int c = 0; c < 3; ++c) w[c] = p->amp_rot * (2.0 * u24(r[1 + c]) - 1.0);
        quat_from_rotvec(w, qw);
        quat_mul(qw, pose + 3, q);
        quat_normalize(q);
        for (int c = 0; c < 4; ++c) cand[3 + c] = q[c];
    } else {
        int k = (int)(((uint64_t)r[1] * (uint32_t)T) >> 32);
        cand[7 + k] = PI * (2.0 * u24(r[2]) - 1.0);
    }
    return kind;
}

double orc_mc_uniform(uint64_t seed, uint32_t system, uint32_t copy, uint32_t step)
{
    uint32_t r[4];
    draw(seed, system, copy, step, 1, r);
    return u24(r[0]);
}

double orc_search_copy(const orc_params *p, const orc_grid *g, const orc_ligand *L,
                       int steps, int cap, uint64_t seed, uint32_t system, uint32_t copy,
                       const double *init_pose, double *best_pose,
                       double *trace_pose, orc_step_rec *trace, orc_step_rec *init_rec)
{
    const int np_ = 7 + L->T;
    double *cur = (double *)malloc(sizeof(double) * np_);
    double *c0 = (double *)malloc(sizeof(double) * np_);
    double *c1 = (double *)malloc(sizeof(double) * np_);
    int it, ne;
    double e_cur = orc_local_opt(p, g, L, cap, init_pose, cur, &it, &ne);
    if (init_rec) { init_rec->e_cur = 0; init_rec->e_cand = e_cur; init_rec->u = 0; init_rec->accept = 1; init_rec->iters = it; init_rec->evals = ne; }
    double e_best = e_cur;
    memcpy(best_pose, cur, sizeof(double) * np_);
    for (int s = 0; s < steps; ++s) {
        if (trace_pose) memcpy(trace_pose + (int64_t)s * np_, cur, sizeof(double) * np_);
        orc_mc_perturb(p, L->T, seed, system, copy, (uint32_t)s, cur, c0);
        double e_c = orc_local_opt(p, g, L, cap, c0, c1, &it, &ne);
        double u = orc_mc_uniform(seed, system, copy, (uint32_t)s);
        int accept = (e_c < e_cur) || (u < exp((e_cur - e_c) / p->t_mc));
        if (trace) { trace[s].e_cur = e_cur; trace[s].e_cand = e_c; trace[s].u = u; trace[s].accept = accept; trace[s].iters = it; trace[s].evals = ne; }
        if (accept) { memcpy(cur, c1, sizeof(double) * np_); e_cur = e_c; }
        if (e_cur < e_best) { e_best = e_cur; memcpy(best_pose, cur, sizeof(double) * np_); }
    }
    free(cur); free(c0); free(c1);
    return e_best;
}

int64_t orc_search(const orc_params *p, const orc_grid *g, const orc_ligand *L,
                   int copies, int steps, int cap, uint64_t seed, uint32_t system,
                   const double *init_poses, double *best_pose, double *best_e,
                   double *trace_pose, orc_step_rec *trace, orc_step_rec *init_rec)
{
    const int np_ = 7 + L->T;
    int64_t total = 0;
#pragma omp parallel for schedule(dynamic, 1) reduction(+ : total)
    for (int c = 0; c < copies; ++c) {
        orc_step_rec *tr = trace ? trace + (int64_t)c * steps : NULL;
        orc_step_rec ir;
        best_e[c] = orc_search_copy(p, g, L, steps, cap, seed, system, (uint32_t)c,
                                    init_poses + (int64_t)c * np_, best_pose + (int64_t)c * np_,
                                    trace_pose ? trace_pose + (int64_t)c * steps * np_ : NULL, tr, &ir);
        if (init_rec) init_rec[c] = ir;
        total += ir.evals;
        if (tr) for (int s = 0; s < steps; ++s) total += tr[s].evals;
    }
    return total;
}

/* Teacher-forced replay of recorded MC steps (parity level 3'): for record k the current pose
 * before the step is given (pre_pose [n][7+T], any implementation's); the oracle evaluates it, draws the
 * perturbation of (system, copy[k], step[k]), relaxes the candidate and takes the Metropolis decision with its own
 * numbers.  OpenMP over records.  Outputs per record: e_cur, cutoff margin of the pre-step pose, kind, e_cand, u,
 * accept, iters, evals (all nullable). */
void orc_replay_steps(const orc_params *p, const orc_grid *g, const orc_ligand *L, int cap, uint64_t seed,
                      uint32_t system, int64_t n, const double *pre_pose, const int32_t *copy, const int32_t *step,
                      double *e_cur, double *cur_cutoff_margin, int32_t *kind, double *e_cand, double *u,
                      int32_t *accept, int32_t *iters, int32_t *evals)
{
    const int np_ = 7 + L->T;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t k = 0; k < n; ++k) {
        double *c0 = (double *)malloc(sizeof(double) * np_), *c1 = (double *)malloc(sizeof(double) * np_);
        orc_diag dg;
        const double ec = orc_eval(p, g, L, pre_pose + k * np_, NULL, NULL, &dg);
        const int kd = orc_mc_perturb(p, L->T, seed, system, (uint32_t)copy[k], (uint32_t)step[k], pre_pose + k * np_, c0);
        int it, ne;
        const double en = orc_local_opt(p, g, L, cap, c0, c1, &it, &ne);
        const double uu = orc_mc_uniform(seed, system, (uint32_t)copy[k], (uint32_t)step[k]);
        if (e_cur) e_cur[k] = ec;
        if (cur_cutoff_margin) cur_cutoff_margin[k] = dg.cutoff_margin;
        if (kind) kind[k] = kd;
        if (e_cand) e_cand[k] = en;
        if (u) u[k] = uu;
        if (accept) accept[k] = (en < ec) || (uu < exp((ec - en) / p->t_mc));
        if (iters) iters[k] = it;
        if (evals) evals[k] = ne;
        free(c0); free(c1);
    }
}

/* ---------------------------------------------------------------------------------------
 * O10 ranking and greedy RMSD clustering (reading S19).
 * ------------------------------------------------------------------------------------- */
double orc_rmsd(const orc_ligand *L, const double *pose_a, const double *pose_b)
{
    double *xa = (double *)malloc(sizeof(double) * 3 * L->N), *xb = (double *)malloc(sizeof(double) * 3 * L->N);
    orc_coords(L, pose_a, xa);
    orc_coords(L, pose_b, xb);
    double s = 0.0;
    for (int i = 0; i < 3 * L->N; ++i) s += (xa[i] - xb[i]) * (xa[i] - xb[i]);
    free(xa); free(xb);
    return sqrt(s / L->N);
}

int orc_topk(const orc_params *p, const orc_ligand *L, int copies, const double *poses,
             const double *e, int k, double rmsd_min, int32_t *out_idx)
{
    (void)p;
    const int np_ = 7 + L->T;
    int *order = (int *)malloc(sizeof(int) * copies);
    for (int i = 0; i < copies; ++i) order[i] = i;
    /* insertion sort: ascending E, ties -> lower copy index (stable) */
    for (int i = 1; i < copies; ++i) {
        int v = order[i], j = i - 1;
        while (j >= 0 && e[order[j]] > e[v]) { order[j + 1] = order[j]; --j; }
        order[j + 1] = v;
    }
    int kept = 0;
    for (int i = 0; i < copies && kept < k; ++i) {
        int c = order[i], ok = 1;
        for (int m = 0; m < kept; ++m)
            if (orc_rmsd(L, poses + (int64_t)c * np_, poses + (int64_t)out_idx[m] * np_) < rmsd_min) { ok = 0; break; }
        if (ok) out_idx[kept++] = c;
    }
    free(order);
    return kept;
}
