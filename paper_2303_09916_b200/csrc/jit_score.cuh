// jit_score.cuh -- run-time specialised score kernel (jit_score.cu): host-side interface used by score.cu.
#pragma once

#include <string>

#include "common.cuh"

#define DOCK_JIT_MAX_ATOMS 40          // forces live in registers (3 per atom): larger ligands use the generic kernel

struct JitOpts {          // all ints: hashed as raw bytes (no padding)
    int want_grad;
    int group;          // chains (duo x partner atom) emitted stage by stage together
    int warps;          // warps per CTA
    int min_blocks;     // __launch_bounds__ second argument (caps the registers)
    int maxrreg;        // --maxrregcount (0 = none)
    int reuse;          // a duo's coordinates loaded for group g are reused by groups g+1 .. g+reuse before being reloaded
    int grid_unroll;    // duos per iteration of the map-lookup loop
    int grid_sets;      // register sets of the map-lookup loop (grid_sets - 1 gathers-in-flight sets ahead of the interpolation)
    int stream;         // 1: pose loads / output stores carry streaming (evict-first) cache hints
    int quad;           // 1: gathers read the 4-corner image dock_grid.quad_dev (two adjacent 16-byte loads); 0: the Cell8 image
    int l2_hint;        // 1: the map gathers carry an L2 evict_last policy
    int prefetch;       // 1: the kinematics loop prefetches every atom's map cell into L2
    int atom_unroll;    // unroll factor of the atom loop of the kinematics
    int sync_every;     // __syncthreads() every this many groups (0 = never): the warps of a CTA share the i-cache window
};

JitOpts jit_default_opts();
bool jit_available();
// DOCK_EINVAL if the ligand / grid is outside what the generator covers (then the caller uses the generic kernel)
int jit_score_source(const dock_params *p, const dock_grid *g, const dock_ligand *L, const JitOpts &o, std::string &out);
int jit_score_launch(const dock_params *p, const dock_grid *g, const dock_ligand *L, const DevParams &P, const DevGrid &G,
                     long long n_poses, const float *poses_dev, float *energy_dev, float *grad_dev, float *terms_dev,
                     cudaStream_t stream);
