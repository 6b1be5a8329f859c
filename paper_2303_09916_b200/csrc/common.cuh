// common.cuh -- device-side descriptors and small helpers shared by the kernels of libdock_b200.
// Product code (sm_100a CUDA).  Shares nothing with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>

#include "../../include/dock.h"

#define FULL_MASK 0xffffffffu

// ---- host-side error plumbing -----------------------------------------------------------------
extern std::atomic<int> g_dock_last_cuda_error;
extern std::atomic<unsigned long long> g_dock_launches;

#define DOCK_CUDA_CHECK(expr)                                   \
    do {                                                        \
        cudaError_t _e = (expr);                                \
        if (_e != cudaSuccess) {                                \
            g_dock_last_cuda_error.store((int)_e);              \
            return DOCK_ECUDA;                                  \
        }                                                       \
    } while (0)

#define DOCK_LAUNCH_CHECK()                                     \
    do {                                                        \
        g_dock_launches.fetch_add(1);                           \
        DOCK_CUDA_CHECK(cudaGetLastError());                    \
    } while (0)

static inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// ---- device descriptors -----------------------------------------------------------------------
// One entry of the gather layout: the 8 corners of the cell whose low corner is node (ix,iy,iz).
//   lo = {G(ix,iy,iz), G(ix+1,iy,iz), G(ix,iy+1,iz), G(ix+1,iy+1,iz)},  hi = the same at iz+1.
// 32 bytes = one L2 sector = one 256-bit load (LDG.E.ENL2.256 on sm_100a): a fully divergent warp
// load costs the L1TEX pipe ~1.8 cycles per lane whatever its width, so one 32-byte load per atom
// halves the gather cost of two 16-byte loads (profiles/r1f.md).
struct __align__(32) Cell8 {
    float4 lo, hi;
};

struct DevParams {
    float w[5];
    float cutoff, cutoff2;
    float k_wall;
    float t_mc;
    float amp_trans, amp_rot;
    float c1, shrink, gtol, curv_eps;
    int   max_trials;
    int   optimizer;           // 0 = BFGS, 1 = Barzilai-Borwein
    float bb_step, bb_fallback;
    // pair term of the thread-per-pose evaluator (eval_thread.cuh), weights folded into the exponents:
    //   A = 8|w1| exp(-(d/0.5)^2) = ex2(cA d^2 + lw1),   B = |w2|/2 exp(-((d-3)/2)^2) = ex2(cB (d-3)^2 + lw2)
    // with sigma = -sign(w1):  sigma dE/dd = d (A + q B) - 3 q B + c4 min(d,0) + wh' [hyd ramp] + whb' [hb ramp]
    // and E = eA sum A + eB sum B + (sigma/2) sum c4 min(d,0)^2 - sigma sum wh' H - 0.7 sigma sum whb' B_hb,
    // where the schedule stores wh' = -sigma w4 and whb' = -sigma w5 / 0.7.  Forces are carried
    // sigma-scaled and multiplied by sigma (exactly, it is +-1) on output.
    float lw1, lw2;            // log2(8|w1|), log2(|w2|/2)  (-inf for a zero weight)
    float sigma;               // -sign(w1)
    float q, m3q;              // sign(w1) sign(w2), -3 q
    float c4;                  // sigma 2 w3
    float eA, eB;              // sign(w1)/8, 2 sign(w2)
};

// Grid maps as the evaluators see them.  Positions are handled relative to a reference node of the
// lattice near its centre (node index ic* on each axis): coordinates stay small, so fp32 keeps
// ~1e-6 A where lab-frame coordinates of 30-50 A would keep ~4e-6 A.
struct DevGrid {
    int   nx, ny, nz;
    int   icx, icy, icz;            // index of the reference node
    float rx, ry, rz;               // fp32 position of the reference node ...
    float rdx, rdy, rdz;            // ... and the remainder (true - fp32) of that position
    float lo_x, lo_y, lo_z;         // -ic*            (cell units, relative to the reference node)
    float hi_x, hi_y, hi_z;         // n-1-ic*
    float h, inv_h, inv_h_lo;       // spacing; fl(1/h) and 1/h - fl(1/h)
    float kw_g, kw_e;               // wall: 2 k h (gradient per cell of overshoot), k h^2
    int   channels, chan_stride;    // 1, or 4 (eq. 4: score, d/dx, d/dy, d/dz at chan_stride entries apart)
    const Cell8  *packed;           // [n_maps][nz][ny][nx] gather layout: the 8 corners of a cell in one 32-byte entry (see dock.h)
    const float  *data;             // [n_maps][nz][ny][nx]
};

// ---- warp-per-pose evaluator (search kernels): compiled ligand in the caller's workspace --------
// One scheduled intra-ligand pair.  ij = i | (j << 16), or -1 for an idle lane (rsum = TPP_MASKED_RSUM).
struct __align__(16) PairRec {
    int   ij;
    float rsum;   // R_i + R_j
    float wh;     // wh'  = -sigma w4 if both hydrophobic else 0        (DevParams)
    float whb;    // whb' = -sigma w5 / 0.7 if donor/acceptor pair else 0
};

struct DevLigand {
    int N, T, P, n_rounds;
    int n_pad;                 // stride of the per-warp coordinate arrays
    const float4  *atom_ref;   // [N] reference xyz relative to the pivot; w = bitcast(map offset in packed entries)
    const int2    *atom_topo;  // [N] {fragment, mask of torsions on the path to the root}
    const float4  *tors_axis;  // [T] unit axis in the reference frame
    const float4  *tors_pt;    // [T] reference position of atom b relative to the pivot; w = bitcast(parent fragment)
    const int2    *tors_ab;    // [T] {a, b}
    const PairRec *sched;      // [n_rounds][32] conflict-free pair schedule
};

struct DevSystem {
    DevGrid   grid;
    DevLigand lig;
    float     box_lo[3], box_size[3];
};

// ---- thread-per-pose evaluator (batch scoring): ligand tables in the kernel-parameter constant
// bank, so that every table read is a uniform constant load and costs no L1 wavefront ------------
#define TPP_TILE 4                      // atoms of the i-tile held in registers in the pair phase
#define TPP_SCHED_QUADS 1600            // capacity of the in-parameter schedule (25.6 KB of 16-byte quads)

// Pair schedule = a stream of 16-byte quads (one uniform 128-bit constant load each).  There is one
// group per tile of TPP_TILE consecutive slots, in slot order, so every atom belongs to exactly one
// group (the evaluator also does the atom's grid lookup there):
//   group   : header {i-slots (4 bytes, byte t = slot of tile atom t; padding repeats slot 0 of the tile),
//                      n2_plain | n1_plain << 8 | n2_hyd << 16 | n1_hyd << 24,
//                      n2_hb | n1_hb << 8 | n_live << 16, 0}
//             then per class (plain, hyd, hb) n2 double records and n1 (0/1) single records.
//   record  : one partner slot j against the 4 tile atoms.  A pair that is not listed gets
//             -(R_i+R_j) = -TPP_MASKED_RSUM: its surface distance is then +1e18 and every term and
//             derivative evaluates to exactly 0 -- no mask test in the instruction stream.
//             class plain: no pair of the record has a hydrophobic or H-bond term; hyd: some pair has
//             the hydrophobic term, none the H-bond term; hb: some pair has the H-bond term.
//     single : {j, 0, 0, 0} {-rsum[4]} [{wh'[4]}  (hyd, hb)] [{whb'[4]}  (hb)]      (the NEGATED radius sum: d = r + (-rsum))
//     double : {jA, jB, 0, 0} then the single-record payload of A, then that of B
//   j is stored as the byte offset of the slot's z column (j * 128); the (x,y) column is at twice that.
//   wh' = -sigma w4 or 0, whb' = -sigma w5 / 0.7 or 0 per pair (see DevParams).
#define TPP_MASKED_RSUM (-1.0e18f)

struct TppLigand {
    int N, T, n_groups, sched_in_param;
    int fm_alias, pad_[3];                  // fragment sums alias consumed force slots (eval_thread.cuh)
    float4 atom_ref[DOCK_MAX_ATOMS];        // slot order (sorted by fragment): xyz rel. pivot, w = bitcast(map offset in entries)
    float4 tors_axis[DOCK_MAX_TORSIONS];    // reference-frame unit axis; w = bitcast(parent fragment)
    float4 tors_pt[DOCK_MAX_TORSIONS];      // reference position of atom b rel. pivot; w = 1 / |ref_b - ref_a|
    unsigned char  tors_a[DOCK_MAX_TORSIONS], tors_b[DOCK_MAX_TORSIONS];   // slots of the axis atoms
    unsigned char  frag_end[DOCK_MAX_TORSIONS + 4];                        // one past the last slot of fragment f
    const uint4 *sched_global;              // the same stream in global memory (used when it does not fit below)
    uint4 sched[TPP_SCHED_QUADS];
};

// ---- device helpers ---------------------------------------------------------------------------
// (forceinline on purpose: as __noinline__ functions -- ~25 call sites, 1700 of the search kernels' 7600 instructions --
// the kernels shrink to 6700 instructions but run 10 % slower, profiles/r2c.md)
__device__ __forceinline__ float warp_sum(float v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(FULL_MASK, v, o);
    return v;
}
__device__ __forceinline__ double warp_sum_d(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(FULL_MASK, v, o);
    return v;
}
__device__ __forceinline__ void ldg_cell(const Cell8 *p, float4 &lo, float4 &hi)
{
    unsigned long long a, b, c, d;
    asm("ld.global.nc.v4.b64 {%0,%1,%2,%3}, [%4];" : "=l"(a), "=l"(b), "=l"(c), "=l"(d) : "l"(p));
    lo.x = __uint_as_float((unsigned)a); lo.y = __uint_as_float((unsigned)(a >> 32));
    lo.z = __uint_as_float((unsigned)b); lo.w = __uint_as_float((unsigned)(b >> 32));
    hi.x = __uint_as_float((unsigned)c); hi.y = __uint_as_float((unsigned)(c >> 32));
    hi.z = __uint_as_float((unsigned)d); hi.w = __uint_as_float((unsigned)(d >> 32));
}
// ---- packed fp32x2 arithmetic (sm_100: FFMA2 / FADD2 / FMUL2) ------------------------------------
// Two IEEE fp32 operations in ONE issue slot (the FMA pipe still spends two cycles): the thread-per-pose
// evaluator is bound by issue slots, not by the FMA pipe, so its pair arithmetic runs on register pairs
// (profiles/r1j.md).  Scalars, immediates and uniform registers broadcast for free in SASS.
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk2(float lo, float hi)
{
    f32x2 r;
    asm("mov.b64 %0, {%1,%2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ f32x2 bc2(float v) { return pk2(v, v); }
__device__ __forceinline__ void up2(f32x2 v, float &lo, float &hi) { asm("mov.b64 {%0,%1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ float sum2(f32x2 v) { float a, b; up2(v, a, b); return a + b; }
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c)
{
    f32x2 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b)
{
    f32x2 d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b)
{
    f32x2 d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ f32x2 sub2(f32x2 a, f32x2 b)
{
    f32x2 d;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}

__device__ __forceinline__ float fast_ex2(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float fast_rsqrt(float x)
{
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// Philox4x32-10 (Salmon et al., SC'11).  counter = (copy, step, slot, system), key = seed lo/hi.
__host__ __device__ inline void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              uint32_t k0, uint32_t k1, uint32_t out[4])
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const unsigned long long p0 = 0xD2511F53ull * (unsigned long long)c0;
        const unsigned long long p1 = 0xCD9E8D57ull * (unsigned long long)c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
        c0 = n0;
        c2 = n2;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

