/*
 * dock_oracle.h -- CPU ORACLE for the DSDP docking-stage hot path (arxiv 2303.09916).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference leg may build, load or call it.
 * It is a plain, slow, double-precision restatement of what the path computes, written
 * from PAPER.md (and the readings listed in DESIGN.md / SURVEY.md 8(c)); it shares no
 * code, header, table or constant generator with the CUDA library under
 * paper_2303_09916_b200/ and neither includes the other.
 *
 * Passages followed (PAPER.md line numbers):
 *   O1  pair potential f_ij            : PAPER.md:49 ("same scoring function" as Vina), eq. s_i = sum_j f_ij at 196
 *   O2  per-type grid maps             : PAPER.md:51 ("every vertex ... summation ... within the cutoff"), eq. 2 at 198-199
 *   O3  pose -> coordinates            : flexible ligand of PAPER.md:49,65 (torsion tree; reading S11)
 *   O4  trilinear E (eq. 2, 198-207) and its partial derivatives (eq. 3, 213-219); wall: PAPER.md:85 (reading S7)
 *   O5  intra-ligand pair terms        : PAPER.md:49
 *   O6  chain rule to force/torque/torsion derivatives
 *   O8  BFGS local optimisation        : PAPER.md:53 (Vina's BFGS, ref. 36 at 183) -- constants are readings (S12): PARITY UNPINNED for the constants
 *   O8' Barzilai-Borwein local optimisation : PAPER.md:53 ("only needs a vector inner product ... no line search"), ref. 37 at 184;
 *       step rule and safeguards are readings (S13): PARITY UNPINNED for the constants, algorithm pinned on quadratics
 *   O9  many-copy Monte-Carlo          : PAPER.md:65-67 (reading S14-S16); search outcome: PARITY UNPINNED beyond GPU-vs-oracle
 *   O10 ranking + RMSD clustering      : PAPER.md:67, 81 (reading S19)
 *   NEXT-2 eq. 4 gradient maps         : PAPER.md:51, 221 -- orc_build_grid_grad + interpolation in orc_eval when orc_grid.gdata != NULL
 *   NEXT-3 site-restrained start poses : Fig. 3 (reading S22) -- orc_init_pose_site
 *   Philox4x32-10                      : Salmon et al. SC'11, as restated in SURVEY.md 8(c) R-rules
 *
 * Units: Angstrom, kcal/mol, radians.  All arrays C-contiguous, host memory, double / int32.
 * pose = [t(3), q(w,x,y,z), theta(T)]   (7+T doubles)
 * grad = [dE/dt(3), torque(3) (lab frame, about the pivot t), dE/dtheta(T)]   (6+T doubles)
 */
#ifndef DOCK_ORACLE_H
#define DOCK_ORACLE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ORC_MAX_TYPES 32

typedef struct {
    int    n_types;
    double radius[ORC_MAX_TYPES];
    int    hydrophobic[ORC_MAX_TYPES];
    int    donor[ORC_MAX_TYPES];
    int    acceptor[ORC_MAX_TYPES];
    double w[5];            /* gauss1, gauss2, repulsion, hydrophobic, hbond */
    double cutoff;          /* 8 A, strict r < cutoff (S3) */
    double k_wall;          /* quadratic wall constant (S7) */
    double t_mc;            /* Metropolis temperature (S15) */
    double amp_trans;       /* translation amplitude per axis (S14) */
    double amp_rot;         /* rotation-vector amplitude per component (S14) */
    double bfgs_c1;         /* Armijo constant */
    double bfgs_shrink;     /* backtracking factor */
    int    bfgs_max_trials; /* line-search trials per iteration */
    double bfgs_gtol;       /* stop when ||g||_2 < gtol */
    double bfgs_curv_eps;   /* skip the update if y.s <= eps*||s||*||y|| */
    double cluster_rmsd;    /* O10 */
    int    topk;            /* O10 */
    int    optimizer;       /* 0 = BFGS (O8), 1 = Barzilai-Borwein (O8'; reading S13) */
    double bb_step;         /* O8': length of the first step and cap on every step, pose units (A / rad) */
    double bb_fallback;     /* O8': step length used when s.y is not safely positive */
} orc_params;

typedef struct {
    int N, T, P;
    const double *ref;          /* [N][3] */
    const int32_t *type;        /* [N] */
    const int32_t *frag;        /* [N], 0 = root */
    const int32_t *tors_parent; /* [T] parent fragment of fragment k+1 (<= k) */
    const int32_t *tors_a;      /* [T] axis atom in the parent fragment */
    const int32_t *tors_b;      /* [T] axis atom in fragment k+1 */
    const int32_t *pairs;       /* [P][2] */
} orc_ligand;

typedef struct {
    int    dims[3];             /* nx, ny, nz */
    double origin[3];
    double h;
    int    n_maps;
    int    type_to_map[ORC_MAX_TYPES]; /* -1 = absent */
    const double *data;         /* [n_maps][nz][ny][nx] */
    const double *gdata;        /* NEXT-2 (eq. 4): [n_maps][3][nz][ny][nx] analytic gradient of the vertex score at the vertices, or NULL:
                                 * then the gradient is that of the interpolant (eq. 3) */
} orc_grid;

/* per-evaluation diagnostics filled by orc_eval when `diag` != NULL */
typedef struct {
    double face_margin;   /* min over atoms/axes of the distance (A) to the nearest cell face or box face */
    double kink_margin;   /* min over intra pairs of |r-cutoff| and of |d - kink| for the active piecewise terms */
    double cutoff_margin; /* min over intra pairs of |r-cutoff| alone: the only place where E itself jumps */
    int    pairs_in_range;/* number of intra pairs with r < cutoff */
    int    atoms_outside; /* atoms with at least one clamped axis */
} orc_diag;

void   orc_default_params(orc_params *p);

/* O1: f(t1,t2,r) and df/dr.  r >= cutoff -> 0. */
double orc_pair(const orc_params *p, int t1, int t2, double r, double *dfdr);

/* Philox4x32-10 */
void   orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);

/* grid geometry: n = round(size/h)+1, origin = center - size/2 */
void   orc_grid_geometry(const double center[3], const double size[3], double h, int dims[3], double origin[3]);

/* O2: brute-force maps.  G is [n_lig_types][nz][ny][nx].  An atom counts iff r < cutoff, decided in double (S3). */
void   orc_build_grid(const orc_params *p, int np, const double *pxyz, const int32_t *ptype,
                      const int dims[3], const double origin[3], double h,
                      int n_lig_types, const int32_t *lig_types, double *G);
/* diagnostic (changes no result): flags[node] = 1 iff some atom lies within `margin` of that node's cutoff sphere;
 * the vertex score jumps there (S3), so the parity tests exempt these nodes and assert they are few.  Returns the count. */
int64_t orc_grid_cutoff_flags(int np, const double *pxyz, const int dims[3], const double origin[3], double h,
                              double cutoff, double margin, uint8_t *flags);
/* NEXT-2 ("we further used the gradient of score obtained by trilinear interpolation", eq. 4 at 221): the
 * gradient of the vertex score at the vertices, GD[t][c][m] = sum_j f'(r) (m - r_j)_c / r over the same atoms as G. */
void orc_build_grid_grad(const orc_params *p, int np, const double *pxyz, const int32_t *ptype,
                         const int dims[3], const double origin[3], double h,
                         int n_lig_types, const int32_t *lig_types, double *GD);

/* O3 */
void   orc_coords(const orc_ligand *L, const double *pose, double *x);

/* O4-O7.  terms = {E_grid, E_wall, E_intra}; grad may be NULL; diag may be NULL. */
double orc_eval(const orc_params *p, const orc_grid *g, const orc_ligand *L,
                const double *pose, double terms[3], double *grad, orc_diag *diag);

/* batch of poses [n][7+T] (OpenMP over poses). E [n]; grad [n][6+T] or NULL; terms [n][3] or NULL; diag [n] or NULL */
void   orc_score_batch(const orc_params *p, const orc_grid *g, const orc_ligand *L, int64_t n,
                       const double *poses, double *E, double *grad, double *terms, orc_diag *diag);
/* diagnostic: conditioning scale A[n][6+T] of each gradient component (sum of |terms|); no result depends on it */
void   orc_grad_cond(const orc_params *p, const orc_grid *g, const orc_ligand *L, const double *pose, double *A);
void   orc_grad_cond_batch(const orc_params *p, const orc_grid *g, const orc_ligand *L, int64_t n,
                           const double *poses, double *A);

/* x (+) s : t += s[0:3]; q <- normalize(quat(rotvec s[3:6]) * q); theta += s[6:] */
void   orc_pose_add(int T, const double *pose, const double *s, double *out);

/* O8 generic core: minimise fn over x with retraction add; n = tangent dim, np_ = len(x).
 * fn(ctx, x, grad) -> f;  add(ctx, x, s, out): out = x (+) s;  obs(ctx, it, f, H[n*n], s, y, updated). */
typedef double (*orc_objective_fn)(void *ctx, const double *x, double *grad);
typedef void   (*orc_retract_fn)(void *ctx, const double *x, const double *s, double *out);
typedef void   (*orc_observer_fn)(void *ctx, int it, double f, const double *H, const double *s, const double *y, int updated);

/* why a local optimisation ended */
#define ORC_EXIT_GTOL       1   /* ||g||_2 < gtol */
#define ORC_EXIT_CAP        2   /* iteration cap reached */
#define ORC_EXIT_LINESEARCH 3   /* no acceptable trial in bfgs_max_trials backtracking steps */
#define ORC_MAX_TRIALS     64

/* decision scalars of one O8 iteration (diagnostic; filled by orc_bfgs / orc_bfgs_step) */
typedef struct {
    int    status;      /* 0 = step accepted, else ORC_EXIT_GTOL / ORC_EXIT_LINESEARCH */
    int    reset;       /* g.d >= 0: H was reset to the identity */
    int    fresh_in, fresh_out;   /* "H is the identity" flag before / after the iteration */
    int    trials;      /* evaluations spent in the line search */
    int    updated;     /* inverse-Hessian update applied (curvature guard passed) */
    double f, gnorm, gp, alpha0, alpha, f_new;
    double armijo_margin[ORC_MAX_TRIALS];  /* (f_trial - f) - c1 alpha g.d of every trial: <= 0 accepts */
    double curv_margin; /* y.s - curv_eps |s| |y|: > 0 updates */
    double min_cutoff_margin; /* orc_bfgs_step only: min over the state and all trial poses of the distance (A) of any
                               * intra pair to the cutoff, where E itself jumps (S3) */
} orc_iter_rec;

/* recs (nullable, capacity max_recs) receives one record per iteration started; exit_reason nullable */
double orc_bfgs(const orc_params *p, int n, int np_, int cap, const double *x0,
                orc_objective_fn fn, orc_retract_fn add, void *ctx,
                double *x_out, int *iters, int *evals, orc_observer_fn obs, void *obs_ctx,
                int *exit_reason, orc_iter_rec *recs, int max_recs);
/* decision scalars of one O8' iteration (diagnostic; filled by orc_bb_step) */
typedef struct {
    int    status;      /* 0 = step taken, ORC_EXIT_GTOL = stopped before it */
    int    branch;      /* 0 = first step (bb_step/|g|), 1 = BB1 s.s/s.y, 2 = fallback bb_fallback/|g| */
    int    capped;      /* step length clipped to bb_step */
    int    pad_;
    double f, gnorm, alpha, f_new;
    double sy_margin;   /* s.y - curv_eps |s| |y|: > 0 takes the BB1 step */
    double cap_margin;  /* alpha |g| - bb_step before clipping: > 0 clips */
    double min_cutoff_margin; /* as in orc_iter_rec */
} orc_bb_rec;

/* O8': x_{k+1} = x_k (+) (-alpha_k g_k), alpha_0 = bb_step/|g|, alpha_k = s.s/s.y (BB1) when
 * s.y > curv_eps |s||y| else bb_fallback/|g|, every step capped at length bb_step; one evaluation per iteration,
 * no line search; returns the best point seen (the method is non-monotone).  Same signature as orc_bfgs. */
double orc_bb(const orc_params *p, int n, int np_, int cap, const double *x0,
                orc_objective_fn fn, orc_retract_fn add, void *ctx,
                double *x_out, int *iters, int *evals, orc_observer_fn obs, void *obs_ctx, int *exit_reason);

/* O8 on the docking objective.  Returns the final energy. */
double orc_local_opt(const orc_params *p, const orc_grid *g, const orc_ligand *L, int cap,
                     const double *pose_in, double *pose_out, int *iters, int *evals);
/* same, also reporting why it ended and (BFGS only; nullable) the per-iteration decision records */
double orc_local_opt_ex(const orc_params *p, const orc_grid *g, const orc_ligand *L, int cap,
                        const double *pose_in, double *pose_out, int *iters, int *evals, int *exit_reason,
                        orc_iter_rec *recs, int max_recs);
/* OpenMP over poses: poses [n][7+T] -> out_pose [n][7+T], out_e [n], out_info [n][3] = (iters, evals, exit reason) */
void   orc_local_opt_batch(const orc_params *p, const orc_grid *g, const orc_ligand *L, int cap, int64_t n,
                           const double *poses, double *out_pose, double *out_e, int32_t *out_info);
/* ONE O8 iteration on the docking objective from a GIVEN state (x, optional gradient g_in at x, H [n][n], fresh);
 * every energy (and the gradient if g_in is NULL) is evaluated here in double.  For the iteration-level
 * teacher-forced parity test.  x_new / H_new nullable. */
int    orc_bfgs_step(const orc_params *p, const orc_grid *g, const orc_ligand *L,
                     const double *x, const double *g_in, const double *H, int fresh, orc_iter_rec *rec,
                     double *x_new, double *H_new);
void   orc_bfgs_step_batch(const orc_params *p, const orc_grid *g, const orc_ligand *L, int64_t n_states,
                           const double *x, const double *g_in, const double *H, const int32_t *fresh,
                           orc_iter_rec *recs, double *x_new, double *H_new);

/* S16 initial pose for (system, copy) from Philox, rounded once to fp32 */
void   orc_init_pose(const double box_center[3], const double box_size[3], int T,
                     uint64_t seed, uint32_t system, uint32_t copy, double *pose);
/* NEXT-3: translation restrained to box ∩ union of balls around the site points (reading S22) */
void   orc_init_pose_site(const double box_center[3], const double box_size[3], int T,
                          uint64_t seed, uint32_t system, uint32_t copy,
                          int n_site, const double *site_xyz, double radius, double *pose);

/* O9 perturbation of MC step `step` of (system, copy): writes the candidate start pose, returns kind (0,1,2) */
int    orc_mc_perturb(const orc_params *p, int T, uint64_t seed, uint32_t system, uint32_t copy,
                      uint32_t step, const double *pose, double *cand);
/* accept uniform of that step */
double orc_mc_uniform(uint64_t seed, uint32_t system, uint32_t copy, uint32_t step);

typedef struct {
    double e_cur;    /* energy of the current pose before the step */
    double e_cand;   /* energy after local optimisation of the candidate */
    double u;        /* accept uniform */
    int    accept;
    int    iters;
    int    evals;
} orc_step_rec;

/* O9 for one copy.  init_pose: [7+T].  Outputs: best_pose [7+T], returns best E.
 * trace_pose [steps][7+T] (pre-step current pose) and trace [steps] may be NULL.
 * init_rec (may be NULL) receives iters/evals/e_cand of the initial local optimisation. */
double orc_search_copy(const orc_params *p, const orc_grid *g, const orc_ligand *L,
                       int steps, int cap, uint64_t seed, uint32_t system, uint32_t copy,
                       const double *init_pose, double *best_pose,
                       double *trace_pose, orc_step_rec *trace, orc_step_rec *init_rec);

/* all copies (OpenMP over copies).  init_poses [copies][7+T]; best_pose [copies][7+T]; best_e [copies];
 * trace_pose [copies][steps][7+T] / trace [copies][steps] / init_rec [copies] nullable; returns total evals */
int64_t orc_search(const orc_params *p, const orc_grid *g, const orc_ligand *L,
                   int copies, int steps, int cap, uint64_t seed, uint32_t system,
                   const double *init_poses, double *best_pose, double *best_e,
                   double *trace_pose, orc_step_rec *trace, orc_step_rec *init_rec);

/* ONE O8' (Barzilai-Borwein) iteration on the docking objective from a GIVEN state (x, optional gradient, previous
 * step s_prev / y_prev unless `first`); energies evaluated here in double.  Iteration-level parity of NEXT-1. */
int    orc_bb_step(const orc_params *p, const orc_grid *g, const orc_ligand *L, const double *x, const double *g_in,
                   const double *s_prev, const double *y_prev, int first, orc_bb_rec *rec, double *x_new);
void   orc_bb_step_batch(const orc_params *p, const orc_grid *g, const orc_ligand *L, int64_t n_states,
                         const double *x, const double *g_in, const double *s_prev, const double *y_prev,
                         const int32_t *first, orc_bb_rec *recs, double *x_new);

/* teacher-forced replay of recorded MC steps (parity level 3'): see dock_oracle.c.  OpenMP over records. */
void   orc_replay_steps(const orc_params *p, const orc_grid *g, const orc_ligand *L, int cap, uint64_t seed,
                        uint32_t system, int64_t n, const double *pre_pose, const int32_t *copy, const int32_t *step,
                        double *e_cur, double *cur_cutoff_margin, int32_t *kind, double *e_cand, double *u,
                        int32_t *accept, int32_t *iters, int32_t *evals);

/* heavy-atom RMSD between two poses, atom order as given, no symmetry correction */
double orc_rmsd(const orc_ligand *L, const double *pose_a, const double *pose_b);

/* O10: returns the number kept (<= k).  out_idx [k] = copy indices in rank order. */
int    orc_topk(const orc_params *p, const orc_ligand *L, int copies, const double *poses,
                const double *e, int k, double rmsd_min, int32_t *out_idx);

int    orc_num_threads(void);
/* diagnostic switch (default off = negative): the objective seen by the optimizers is rounded to a (24 - drop_bits)-bit
 * significand -- see dock_oracle.c */
void   orc_diag_round_eval_fp32(int drop_bits);

#ifdef __cplusplus
}
#endif
#endif
