/*
 * dock.h -- C-ABI of the B200-native docking hot path of DSDP (arxiv 2303.09916).
 *
 * ONE thing lives behind this header: the data-parallel hot path of DSDP's docking stage
 * (Appendix): per-type grid maps of the Vina-style pair
 * potential, fused pose -> coordinates -> trilinear energy + analytic gradient, an on-device
 * many-copy Monte-Carlo search with a BFGS local optimizer, and top-k + RMSD clustering.
 * All of it runs in hand-written sm_100a CUDA kernels; there is no CPU fallback.
 *
 * Conventions:
 *  - Plain C, no exceptions.  Every function returns an int status: DOCK_OK (0) or a negative code.
 *  - The library OWNS NOTHING on the device: grids, poses, outputs and the scratch workspace are
 *    allocated by the caller and passed as raw device pointers ("_dev").  Small topology /
 *    parameter structs are HOST pointers; they are validated, compiled and copied into the
 *    workspace by the call and may be freed as soon as the call returns.
 *  - All work is enqueued on the caller's stream (`stream` is a cudaStream_t passed as void*;
 *    NULL = the legacy default stream).  The *_dev entry points never synchronise the device.
 *    The *_host entry points take host buffers, copy in/out on `stream` and synchronise that
 *    stream before returning.
 *  - Workspace protocol: if `ws_bytes` is smaller than required (or ws_dev is NULL) the call does
 *    no work, writes the requirement to *needed (if non-NULL) and returns DOCK_EWORKSPACE.
 *  - Units: Angstrom, kcal/mol, radians.  Arrays are C-contiguous, fp32 / int32 unless stated.
 *  - pose = [t(3), q(w,x,y,z), theta(T)] (7+T floats); t is the position of the pivot (centroid
 *    of the root-fragment reference atoms), q the orientation (normalised on read).
 *    grad = [dE/dt(3), torque(3) (lab frame, about t), dE/dtheta(T)] (6+T floats).
 */
#ifndef DOCK_H
#define DOCK_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define DOCK_MAX_XS_TYPES 32   /* size of the XS type table */
#define DOCK_MAX_TORSIONS 32   /* T <= 32 */
#define DOCK_MAX_ATOMS    128  /* N <= 128 ligand heavy atoms */
#define DOCK_MAX_TOPK     32

#define DOCK_OK          0
#define DOCK_EINVAL     (-1)   /* null pointer, bad size, malformed torsion tree, type without a map ... */
#define DOCK_EWORKSPACE (-2)   /* workspace too small; *needed holds the requirement */
#define DOCK_ECUDA      (-3)   /* a CUDA call failed; see dock_last_cuda_error() */
#define DOCK_ECAPACITY  (-4)   /* dock_topk_fixed only: the ligand needs more than the library's built-in scratch array */

/* Scoring + search parameters.  The paper prints none of them ("the same scoring
 * function" as Vina); dock_default_params() fills the readings S1, S2, S3, S7, S12, S14, S15, S19
 * of SURVEY.md 8(c). */
typedef struct dock_params {
    int32_t n_types;                          /* number of XS type ids in use (17) */
    float   radius[DOCK_MAX_XS_TYPES];        /* XS radius per type id */
    int32_t hydrophobic[DOCK_MAX_XS_TYPES];
    int32_t donor[DOCK_MAX_XS_TYPES];
    int32_t acceptor[DOCK_MAX_XS_TYPES];
    float   w[5];                             /* gauss1, gauss2, repulsion, hydrophobic, hbond */
    float   cutoff;                           /* 8 A; a pair counts iff r < cutoff (the kernels decide it on r^2 in fp32) */
    float   k_wall;                           /* quadratic wall, kcal/mol/A^2 per axis overshoot */
    float   t_mc;                             /* Metropolis temperature, kcal/mol */
    float   amp_trans;                        /* MC translation amplitude per axis, A */
    float   amp_rot;                          /* MC rotation-vector amplitude per component, rad */
    float   bfgs_c1;                          /* Armijo constant */
    float   bfgs_shrink;                      /* backtracking factor */
    int32_t bfgs_max_trials;                  /* line-search trials per iteration */
    float   bfgs_gtol;                        /* stop when ||g||_2 < gtol */
    float   bfgs_curv_eps;                    /* skip the update if y.s <= eps ||s|| ||y|| */
    float   cluster_rmsd;                     /* top-k clustering radius, A (PAPER.md:81 RMSD) */
    int32_t topk;                             /* number of poses to report, <= DOCK_MAX_TOPK */
    int32_t optimizer;                        /* local optimizer: 0 = BFGS + backtracking, 1 = Barzilai-Borwein */
    float   bb_step;                          /* BB: length of the first step and cap on every step (A / rad) */
    float   bb_fallback;                      /* BB: step length when s.y is not safely positive */
    int32_t grad_mode;                        /* grid gradient: 0 = gradient of the interpolant (eq. 3), 1 = interpolated
                                               * per-vertex gradients (eq. 4; NEXT-2).  Read by dock_build_grids,
                                               * which then writes 4 channels per map; the evaluators follow dock_grid.n_channels */
    int32_t search_kernel;                    /* decomposition of dock_search / dock_local_opt_*: 1 = one warp per copy; 2 = one CTA of
                                               * 4 warps per copy -- with BFGS the warps evaluate 4 consecutive backtracking trials of the
                                               * line search at once (bit-identical to 1; only evaluations the sequential line search would
                                               * make are counted), with Barzilai-Borwein (no line search) they share each evaluation (atoms
                                               * over the threads, pair rounds over the warps: results agree with 1 to round-off);
                                               * 0 = chosen by the library: 2 for n_systems x copies <= 512, else 1 */
    int32_t score_kernel;                     /* dock_score_batch[_host]: 0 or 1 = the generic thread-per-pose kernel; 2 = a kernel specialised
                                               * for this ligand, generated and compiled at run time (NVRTC, 0.4-6 s per ligand, cached per
                                               * device / ligand / parameters): DOCK_ECUDA if the compiler is missing, DOCK_EINVAL above 40
                                               * atoms or with eq. 4 maps (it reads dock_grid.quad_dev).  Same arithmetic per pair / atom / torsion; sums are taken in a
                                               * different order */
} dock_params;

/* Search / interpolation box: n_axis = round(size/spacing)+1 nodes,
 * origin = fl32(center - size/2). */
typedef struct dock_box {
    float center[3];
    float size[3];
    float spacing;
} dock_box;

typedef struct dock_protein {   /* HOST arrays */
    int32_t        n;
    const float   *xyz;         /* [n][3] */
    const int32_t *type;        /* [n] XS type ids */
} dock_protein;

/* Flexible ligand as a torsion tree; HOST arrays.  Fragment 0 is the root; torsion k joins
 * fragment tors_parent[k] (<= k) to fragment k+1, rotating fragment k+1 and its descendants by
 * theta_k (right-handed) about the axis ref[tors_a[k]] -> ref[tors_b[k]] (a in the parent
 * fragment, b in fragment k+1).  theta = 0 reproduces ref_xyz. */
typedef struct dock_ligand {
    int32_t        N, T, P;
    const float   *ref_xyz;        /* [N][3] reference conformation */
    const int32_t *type;           /* [N] XS type ids */
    const int32_t *atom_fragment;  /* [N] */
    const int32_t *tors_parent;    /* [T] */
    const int32_t *tors_a;         /* [T] */
    const int32_t *tors_b;         /* [T] */
    const int32_t *pairs;          /* [P][2] intra-ligand scoring pairs, i != j, each unordered pair at most once */
} dock_ligand;

/* Grid-map descriptor written by dock_build_grids.  Two DEVICE images of the same maps live in the
 * caller's buffer (dock_grid_bytes() bytes, 256-byte aligned):
 *   data_dev   [n_maps][nz][ny][nx] fp32 -- the maps themselves: node (ix,iy,iz) at
 *              origin + spacing*(ix,iy,iz) holds eq. 2's vertex score;
 *   packed_dev [n_maps][nz][ny][nx][8] fp32 -- the gather layout read by every evaluator: entry
 *              (ix,iy,iz) = the 8 corners of the cell whose low corner is that node, in the order
 *              {G(ix,iy,iz), G(ix+1,iy,iz), G(ix,iy+1,iz), G(ix+1,iy+1,iz)} then the same four at
 *              iz+1 (indices clamped to the last node), so a cell is ONE aligned 32-byte load
 *              (DESIGN.md "Data layout").  Values are bit-identical copies of data_dev.
 *   quad_dev   the 4-corner image described at the field (single-channel maps only). */
typedef struct dock_grid {
    int32_t      dims[3];                          /* nx, ny, nz */
    float        origin[3];
    float        spacing;
    int32_t      n_maps;
    int32_t      type_to_map[DOCK_MAX_XS_TYPES];   /* XS type id -> map index, -1 = absent */
    const float *data_dev;                         /* DEVICE pointer, caller-owned */
    const float *packed_dev;                       /* DEVICE pointer into the same buffer */
    int32_t      n_channels;                       /* 1: data_dev [n_maps][nz][ny][nx]; 4 (eq. 4): [n_maps][4][nz][ny][nx] with channels
                                                    * (score, d/dx, d/dy, d/dz) -- packed_dev likewise; 0 is read as 1 */
    const float *quad_dev;                         /* DEVICE pointer into the same buffer, or NULL (eq. 4 maps): the 4-corner image
                                                    * [n_maps][ny][nx][nz][4] = {G(ix,iy,iz), G(ix+1,iy,iz), G(ix,iy+1,iz), G(ix+1,iy+1,iz)},
                                                    * z fastest, so the planes iz and iz+1 of a cell are two adjacent 16-byte loads; half
                                                    * the bytes of packed_dev (it fits an L2 half); read by the specialised score kernel */
} dock_grid;

/* Optional per-(system, copy, step) trace of the search; with the stateless Philox counter it
 * is enough to replay any single MC step (teacher-forced parity).
 * One record = DOCK_TRACE_HEADER floats followed by the pre-step pose (7+T_max floats). */
#define DOCK_TRACE_HEADER 8   /* e_cur, e_cand, u, accept, iters, evals, kind, reserved */

/* Why a local optimisation ended (reading S12). */
#define DOCK_EXIT_GTOL       1   /* ||g||_2 < bfgs_gtol */
#define DOCK_EXIT_CAP        2   /* iteration cap reached */
#define DOCK_EXIT_LINESEARCH 3   /* no acceptable trial in bfgs_max_trials backtracking steps */

/* Optional per-iteration trace of the BFGS local optimizer (dock_local_opt_trace): the state each iteration starts
 * from and its decision scalars -- enough to redo that single iteration elsewhere (iteration-level teacher-forced
 * parity).  One record = DOCK_ITER_HEADER floats
 *   {f, |g|, g.d, alpha0, alpha (last tried), f_new (last trial), status (0 = step taken, else DOCK_EXIT_*),
 *    trials (evaluations of the line search), updated (inverse Hessian updated), reset (H reset to I: g.d >= 0),
 *    fresh_in, fresh_out ("H is the identity" before / after)}
 * followed by the pose x[7+T], the gradient g[6+T] at x and the inverse Hessian H[(6+T)^2] (row-major) the iteration
 * starts from.  With the Barzilai-Borwein optimizer (params->optimizer = 1) the header holds
 *   {f, |g|, 0, 0, alpha, f_new, status, branch (0 = first step, 1 = s.s/s.y, 2 = fallback), 0, capped, 0, 0}
 * and the H area starts with the previous step s[6+T] and gradient change y[6+T] (zeros at iteration 0). */
#define DOCK_ITER_HEADER 12

/* ---- parameters ----------------------------------------------------------------------------- */
int dock_default_params(dock_params *out);

/* ---- A1: grid maps ----------------------------------------
 * G[m][node] = sum over protein atoms j with |node - r_j| < cutoff of f(lig_types[m], type_j, r).
 * protein: host.  grid_dev: device, 256-byte aligned, grid_bytes >= dock_grid_bytes(params, box, n_lig_types)
 * (checked: DOCK_EINVAL if the buffer is too small -- with grad_mode = 1 the maps have 4 channels).
 * out_desc (host) receives the descriptor with data_dev = grid_dev and packed_dev behind it.
 * Errors: DOCK_EINVAL for null pointers, n < 0, spacing <= 0, type ids outside [0, n_types), short or misaligned buffer. */
int dock_grid_dims(const dock_box *box, int32_t dims[3]);
/* bytes of the caller's grid buffer for n_lig_types maps over `box` (both images, all channels of params->grad_mode);
 * 0 on bad input. */
size_t dock_grid_bytes(const dock_params *params, const dock_box *box, int32_t n_lig_types);
int dock_build_grids(const dock_params *params, const dock_protein *protein, const dock_box *box,
                     int32_t n_lig_types, const int32_t *lig_types,
                     float *grid_dev, size_t grid_bytes, dock_grid *out_desc,
                     void *ws_dev, size_t ws_bytes, size_t *needed, void *stream);

/* Batched form (BASELINE.json configs[3]): n_systems (protein, box) pairs with one ligand-type list in ONE upload and
 * ONE pair of launches (build, pack) over all systems.  proteins, boxes, out_descs: HOST arrays [n_systems];
 * grid_dev: HOST array of n_systems DEVICE buffers, grid_bytes: HOST array of their sizes (each checked against
 * dock_grid_bytes).  The workspace holds every system's cell lists: *needed = their sum. */
int dock_build_grids_batch(const dock_params *params, int32_t n_systems, const dock_protein *proteins,
                           const dock_box *boxes, int32_t n_lig_types, const int32_t *lig_types,
                           float *const *grid_dev, const size_t *grid_bytes, dock_grid *out_descs,
                           void *ws_dev, size_t ws_bytes, size_t *needed, void *stream);

/* ---- A2-A5: fused pose -> coordinates -> energy + gradient (eq. 2-3 at 198-219) --
 * poses_dev [n_poses][7+T]; energy_dev [n_poses]; grad_dev [n_poses][6+T] or NULL;
 * terms_dev [n_poses][3] = (E_grid, E_wall, E_intra) or NULL.  E = sum of the three terms. */
int dock_score_batch(const dock_params *params, const dock_grid *grid, const dock_ligand *ligand,
                     int64_t n_poses, const float *poses_dev,
                     float *energy_dev, float *grad_dev, float *terms_dev,
                     void *ws_dev, size_t ws_bytes, size_t *needed, void *stream);

/* Same, with HOST buffers for poses / energy / grad / terms (copies inside the call; pinned memory makes them
 * asynchronous).  The batch is processed in up to 8 chunks through a three-stage pipeline -- host->device copy,
 * kernel, device->host copy -- so that both PCIe directions overlap the arithmetic; the kernels run on `stream`,
 * the copies on two side streams that the library creates once per device (the only resources it owns; calls on
 * the same device from several host threads are serialised by a mutex).  The call returns after everything has
 * completed (`stream` is synchronised once); on an error every copy already enqueued is drained first. */
int dock_score_batch_host(const dock_params *params, const dock_grid *grid, const dock_ligand *ligand,
                          int64_t n_poses, const float *poses_host,
                          float *energy_host, float *grad_host, float *terms_host,
                          void *ws_dev, size_t ws_bytes, size_t *needed, void *stream);

/* ---- A6: BFGS local optimisation of a batch of start poses -----------------------
 * poses_dev [n][7+T] in; out_pose_dev [n][7+T]; out_e_dev [n];
 * out_iters_dev [n][3] = (iterations, evaluations, DOCK_EXIT_* reason) or NULL */
int dock_local_opt_batch(const dock_params *params, const dock_grid *grid, const dock_ligand *ligand,
                         int64_t n_poses, int32_t max_iters, const float *poses_dev,
                         float *out_pose_dev, float *out_e_dev, int32_t *out_iters_dev,
                         void *ws_dev, size_t ws_bytes, size_t *needed, void *stream);
/* Same with the per-iteration trace:
 * iter_trace_dev [n][trace_cap][DOCK_ITER_HEADER + (7+T) + (6+T) + (6+T)^2] floats, one record per iteration STARTED
 * (the last one is the stop itself unless the cap ended the run); iterations >= trace_cap are not recorded.
 * The caller zero-fills the buffer if it wants to tell unused records apart. */
int dock_local_opt_trace(const dock_params *params, const dock_grid *grid, const dock_ligand *ligand,
                         int64_t n_poses, int32_t max_iters, const float *poses_dev,
                         float *out_pose_dev, float *out_e_dev, int32_t *out_iters_dev,
                         float *iter_trace_dev, int32_t trace_cap,
                         void *ws_dev, size_t ws_bytes, size_t *needed, void *stream);

/* ---- S16: initial poses from Philox ("randomly generated within this box", 67) ----
 * Generated on the host in double, rounded once to fp32.  out_host [copies][7+T] = the poses of copies
 * copy_base .. copy_base + copies - 1 of `system` (the Philox counter words, so a shard of copies starts exactly
 * where the same copies of an unsharded run start). */
int dock_init_poses(const dock_box *box, int32_t T, uint64_t seed, uint32_t system, uint32_t copy_base,
                    int32_t copies, float *out_host);

/* ---- NEXT-3: initial poses restrained to the adaptive search space (Fig. 3) ------
 * "A union set of balls with 7 A radius, centered at each discrete points of predicted binding site ... The
 * intersection of this cube and the union set of balls is taken as the space for binding site search.  The
 * initial ligand positions are ... restrained to the searching space."  Reading S22: the
 * translation is drawn uniformly in the box by rejection (Philox slots 0x100 + attempt, 256 attempts, then
 * the site point copy mod n_site); orientation and torsions as dock_init_poses.  site_xyz_host [n_site][3],
 * same frame as the box; out_host [copies][7+T], to be passed to dock_search as init poses after upload. */
int dock_init_poses_site(const dock_box *box, int32_t T, uint64_t seed, uint32_t system, uint32_t copy_base,
                         int32_t copies, int32_t n_site, const float *site_xyz_host, float radius, float *out_host);

/* ---- A6-A8: many-copy Monte-Carlo search + top-k -----------------------------
 * n_systems independent systems in one launch; grids[s], ligands[s], boxes[s] are HOST arrays of
 * descriptors.  T_max = max over systems of T; pose rows are 7+T_max floats wide (unused tail 0).
 * system_base / copy_base: system s, copy c of this call draw the Philox streams of (system_base + s,
 * copy_base + c) -- a multi-GPU run that shards systems or copies passes the index of its
 * first unit and reproduces the unsharded run bit for bit; 0, 0 otherwise.  (One condition: with search_kernel = 0 the
 * kernel is chosen from the size of EACH call.  BFGS gives the same bits on both kernels; Barzilai-Borwein only agrees to
 * round-off between them, so a BB run that must reproduce across shardings sets search_kernel to 1 or 2.)
 * Everything that can be rejected (sizes, shared-memory needs, mixed gradient modes) is rejected before any work is
 * enqueued.
 * init_poses_dev [n_systems][copies][7+T_max] or NULL (then generated by dock_init_poses' rule).
 * best_pose_dev [n_systems][copies][7+T_max]; best_e_dev [n_systems][copies];
 * topk_pose_dev [n_systems][k][7+T_max]; topk_e_dev [n_systems][k]; topk_idx_dev [n_systems][k]
 * (copy index, -1 = unused); topk_count_dev [n_systems]  (k = params->topk)  -- all nullable as a group;
 * trace_dev [n_systems][copies][steps][DOCK_TRACE_HEADER + 7+T_max] or NULL;
 * eval_counter_dev: one uint64, incremented by the number of score+gradient evaluations, or NULL. */
int dock_search(const dock_params *params, int32_t n_systems,
                const dock_grid *grids, const dock_ligand *ligands, const dock_box *boxes,
                int32_t copies, int32_t steps, int32_t bfgs_max_iters, uint64_t seed,
                uint32_t system_base, uint32_t copy_base,
                const float *init_poses_dev,
                float *best_pose_dev, float *best_e_dev,
                float *topk_pose_dev, float *topk_e_dev, int32_t *topk_idx_dev, int32_t *topk_count_dev,
                float *trace_dev, uint64_t *eval_counter_dev,
                void *ws_dev, size_t ws_bytes, size_t *needed, void *stream);

/* ---- A8 alone: rank + greedy RMSD clustering of given poses -----------------
 * poses_dev [n][7+T], e_dev [n] -> out_idx_dev [k], out_count_dev [1]. */
int dock_topk(const dock_params *params, const dock_ligand *ligand, int32_t n,
              const float *poses_dev, const float *e_dev,
              int32_t *out_idx_dev, int32_t *out_count_dev,
              void *ws_dev, size_t ws_bytes, size_t *needed, void *stream);

/* ---- A8 without any device allocation ---------------------------------------
 * dock_topk for callers that cannot allocate device memory, and therefore have no workspace to hand over: a
 * plug-in given raw pointers but no allocator, code inside a region where cudaMalloc / cudaFree are forbidden or
 * would synchronise the device, a loop with a hard latency budget.  Inputs, outputs and results are exactly
 * dock_topk's (same kernel, same tables); only the workspace arguments are gone.  The ligand tables and the system
 * descriptor the kernel reads go into an array of DOCK_TOPK_FIXED_BYTES that is part of the library's device image.
 * What that implies:
 *  - Cost: every GPU that loads libdock_b200.so carries those DOCK_TOPK_FIXED_BYTES until the process exits, used or not.
 *  - Limit: the ligand's tables must fit (*needed, if non-NULL, receives their size; a 60-atom / 15-torsion ligand
 *    with 1483 scoring pairs takes 26 368 bytes).  A larger ligand is refused with DOCK_ECAPACITY before anything is
 *    enqueued or written; use dock_topk with your own workspace for it.  The other limits are dock_topk's.
 *  - The call makes no cudaMalloc, cudaFree or other allocating library call, at any time.
 *  - Set-up: the FIRST call on each device (with that device current) asks the runtime for the array's device
 *    address and keeps it; make that first call outside any stream capture.  Later calls only read the cached address.
 *  - One array per device, shared by every call: calls on the same stream are ordered and safe; calls whose GPU work
 *    can overlap (different streams, different host threads on one device) overwrite each other's tables -- a data race
 *    with undefined results.  Serialise them yourself.  The array keeps the last call's contents between calls;
 *    nothing relies on that: each call rewrites everything its kernel will read.
 * Errors: DOCK_EINVAL as dock_topk; DOCK_ECAPACITY as above; DOCK_ECUDA if the address query or an enqueue fails. */
#define DOCK_TOPK_FIXED_BYTES 65536
int dock_topk_fixed(const dock_params *params, const dock_ligand *ligand, int32_t n,
                    const float *poses_dev, const float *e_dev,
                    int32_t *out_idx_dev, int32_t *out_count_dev, size_t *needed, void *stream);

/* ---- end-to-end convenience with HOST buffers: build grids + search + top-k for one system ----
 * out_topk_pose_host [k][7+T], out_topk_e_host [k], out_count_host [1]; copies H<->D inside. */
int dock_system_host(const dock_params *params, const dock_protein *protein, const dock_box *box,
                     const dock_ligand *ligand, int32_t n_lig_types, const int32_t *lig_types,
                     int32_t copies, int32_t steps, int32_t bfgs_max_iters, uint64_t seed,
                     float *out_topk_pose_host, float *out_topk_e_host, int32_t *out_count_host,
                     uint64_t *out_evals_host,
                     float *grid_dev, size_t grid_bytes, void *ws_dev, size_t ws_bytes, size_t *needed, void *stream);

/* ---- measured roofs --------------------------------------------------
 * Runs four micro-kernels on `stream` (synchronising it) and writes to out_host[4]:
 *   [0] FP32 FMA rate, scalar FFMA, TFLOP/s       [1] the same with packed fp32x2 FMAs (FFMA2), TFLOP/s
 *   [2] MUFU (ex2) rate, T operations/s           [3] fully divergent 32-byte gathers from an L2-resident table, T lanes/s
 * These are the denominators of bench.py's roofline (nothing on this path is bound by HBM or the tensor cores, the two
 * peaks MEASURED_PEAKS.json holds).  ws_dev: 32-byte aligned, *needed bytes (about 16 MB). */
int dock_probe_peaks(float *out_host, void *ws_dev, size_t ws_bytes, size_t *needed, void *stream);

/* ---- diagnostics and measurement: NOT part of the hot-path boundary of SURVEY.md 8(b) ---------
 * (dock_probe_peaks above belongs here too: bench.py divides by its output.) */
/* CUDA source of the ligand-specialised score kernel dock_score_batch would compile for (params, grid, ligand)
 * (score_kernel = 2; A2-A5).  buf: HOST, cap bytes; *needed = length + 1; DOCK_EWORKSPACE if cap is short,
 * DOCK_EINVAL if the ligand is outside what the generator covers.  No device work. */
int dock_score_jit_source(const dock_params *params, const dock_grid *grid, const dock_ligand *ligand,
                          int32_t want_grad, char *buf, size_t cap, size_t *needed);
/* Compiles that source for sm_100a with NVRTC (host only, needs no GPU) and reports the size of the cubin: the "does it build" check
 * of the run-time kernel.  DOCK_ECUDA if NVRTC (libnvrtc.so.12 of CUDA >= 12.9) is missing or the compilation fails. */
int dock_score_jit_compile(const dock_params *params, const dock_grid *grid, const dock_ligand *ligand,
                           int32_t want_grad, size_t *cubin_bytes);
/* The specialised kernels are cached per (device, ligand, parameters, want_grad), at most `limit` per device (default 64):
 * when a device's cache is full the least recently used kernel is unloaded (after a cudaDeviceSynchronize on that device:
 * it may still be running) before the new one is compiled.  new_limit in [1, 65536] sets the limit for later insertions,
 * new_limit < 0 only queries; *old_limit / *entries (nullable) receive the limit before the call and the number of cached
 * kernels over all devices.  DOCK_EINVAL for new_limit = 0 or > 65536. */
int dock_score_jit_cache(int32_t new_limit, int32_t *old_limit, int32_t *entries);
const char *dock_score_jit_log(void);            /* compiler log of the last failed run-time compilation ("" = none) */
int         dock_last_cuda_error(void);          /* cudaError_t of the last failing CUDA call (0 = none) */
const char *dock_version(void);
/* number of kernel launches issued by this library since load (for bench.py's gpu_launches) */
uint64_t    dock_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* DOCK_H */
