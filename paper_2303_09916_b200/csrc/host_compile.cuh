// host_compile.cuh -- host-side "compile" steps: validate the caller's structs and turn them into
// device-ready blobs (no device work here).
#pragma once

#include <vector>

#include "common.cuh"

struct LigandBlob {
    std::vector<unsigned char> bytes;   // device image, 16-byte aligned sections
    DevLigand rel;                      // pointer fields hold BYTE OFFSETS into `bytes`
};

// DOCK_OK or DOCK_EINVAL.  `g` may be NULL (then no type->map lookup is done; map offsets are 0),
// which is what dock_topk uses.
int dock_compile_ligand(const dock_params *p, const dock_grid *g, const dock_ligand *lig, LigandBlob &out);

// Turn the offsets of `b.rel` into pointers relative to `dev_base`.
DevLigand dock_relocate_ligand(const LigandBlob &b, const unsigned char *dev_base);

int dock_validate_params(const dock_params *p);
int dock_make_dev_params(const dock_params *p, DevParams *out);
int dock_make_dev_grid(const dock_params *p, const dock_grid *g, DevGrid *out);

// Thread-per-pose tables (eval_thread.cuh).  DOCK_OK or DOCK_EINVAL.  If the pair schedule does not
// fit TppLigand::sched, out.sched_in_param = 0 and `overflow` holds the stream for the caller to
// upload (then point out.sched_global at it); otherwise `overflow` is empty.
int dock_compile_tpp(const dock_params *p, const dock_grid *g, const dock_ligand *lig, TppLigand &out,
                     std::vector<uint4> &overflow);

// number of floats of per-warp shared memory the warp-per-pose evaluator needs for this ligand
static inline int eval_scratch_floats(int n_pad, int T) { return 8 * n_pad + 2 * ((T + 3) & ~3) + 40 * T; }
