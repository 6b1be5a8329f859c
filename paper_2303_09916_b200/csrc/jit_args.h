// jit_args.h -- the ONE struct shared by the host launcher (jit_score.cu) and the run-time generated,
// ligand-specialised score kernel (its text is pasted in front of the generated source, so both sides always
// agree on the layout).  Plain C types only.
#pragma once

#define DOCK_JIT_STR_(...) #__VA_ARGS__
#define DOCK_JIT_STR(...) DOCK_JIT_STR_(__VA_ARGS__)

// grid geometry (DevGrid, common.cuh) and the buffers of one dock_score_batch call; the pair-term constants
// (DevParams) are literals in the generated text
#define DOCK_JIT_ARGS_BODY                                                                          \
    int nx, ny, nz, icx, icy, icz;                                                                    \
    float rx, ry, rz, rdx, rdy, rdz;                                                                \
    float lo_x, lo_y, lo_z, hi_x, hi_y, hi_z;                                                       \
    float inv_h, inv_h_lo, kw_g, kw_e;                                                              \
    long long map_stride;     /* packed entries between two maps (all channels) */                  \
    const void *packed;       /* Cell8 [n_maps][nz][ny][nx], or the quad image float4 [n_maps][ny][nx][nz] */ \
    long long n_poses;                                                                              \
    const float *poses;                                                                             \
    float *energy, *grad, *terms;

struct JitArgs {
    DOCK_JIT_ARGS_BODY
};
