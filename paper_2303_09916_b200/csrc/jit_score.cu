// jit_score.cu -- ligand-specialised score + gradient kernel, generated and compiled at run time (NVRTC).
//
// SURVEY.md 8(a) A2-A5 (eq. 2-3 at 198-219) for dock_score_batch, selected by dock_params.score_kernel = 2.
// All poses of a batch share ONE ligand, so what the generic thread-per-pose kernel (eval_thread.cuh) decodes at run
// time -- the intra-ligand pair list with its radius sums and term classes -- can be compile-time constants: the pair
// phase becomes straight-line code with no schedule stream, no masked pairs (exactly the listed pairs are evaluated),
// no address arithmetic, and with the per-atom forces in REGISTERS.  Still one THREAD per pose, same arithmetic per
// pair, per atom and per torsion as the generic kernel.
//
// What bounds the design is the instruction cache (measured, profiles/r2b.md): straight-line code runs at full issue
// rate up to 32 KB, at ~3 cycles per instruction per warp up to 128 KB (8192 instructions) and at ~6 beyond.  A
// 30-atom ligand has ~290 pairs at ~19 instructions each, so ONLY the pair phase is unrolled; everything else loops:
//
//   phase 1   A2: loop over fragments and atoms, tables in the constant bank, frames in shared memory.  Coordinates
//             go to shared memory packed by DUO (two atoms that share fp32x2 register pairs): float4 (x0,x1,y0,y1)
//             + float2 (z0,z1).
//   (map image) the gathers read dock_grid.quad_dev, the 4-corner image (68 MB for 81^3 x 8: it fits an L2 half, which the
//             136 MB 8-corner image of the other evaluators does not -- L2 hit rate 78 % against 46 %).
//   phase 2a  A3: loop over duos, 2U atoms per iteration, software-pipelined by one iteration (the 32-byte map
//             gathers of the next atoms are in flight while the current ones are interpolated); sigma-scaled grid
//             forces go to shared memory and seed the force registers.
//   phase 2b  A4: unrolled.  The atoms are matched into duos so that the listed pairs between two duos cover as few
//             CHAINS as possible (148 for the 287 pairs of BASELINE configs[1]): a chain = two pairs in the two lanes
//             of FFMA2 / FADD2 / FMUL2 -- duo x one partner atom (broadcast), duo x duo lane by lane, or any two pairs;
//             a leftover pair runs as scalar code.  Chains are emitted in groups, stage by stage (distances, rsqrt,
//             exponent arguments, ex2, forces).  The cutoff test is dropped for pairs whose distance can never reach
//             the cutoff (triangle inequality along the torsion path).  Coordinates are re-read from shared memory
//             group by group (volatile loads: otherwise the compiler keeps all 3N of them in registers).
//   phases 3 + 4  A5: fragment force / torque sums and the up-sweep over the torsion tree, unrolled (the forces are
//             in registers).
//
// The text is compiled for sm_100a with NVRTC (dlopen'ed: the toolkit's libnvrtc.so.12, CUDA >= 12.9 for the 256-bit
// load), loaded with cudaLibraryLoadData and cached per (device, ligand, parameters).  Measured on B200
// (profiles/r2b.md): 1.15x the generic kernel on configs[1] (N = 30, 7.8 k instructions: the unrolled part runs in the
// 3-cycle regime of the i-cache), 1.3x for ligands of 12-20 atoms, 0.84x at 33 atoms (code > 128 KB), and a
// compilation of 0.4-6 s per ligand -- which is why it is opt-in and the generic kernel stays the default.
#include <dlfcn.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <mutex>
#include <string>
#include <vector>

#include "common.cuh"
#include "host_compile.cuh"
#include "jit_args.h"
#include "jit_score.cuh"

namespace {

// ---- description of the ligand in slot order ------------------------------------------------------
struct JitTors { float ux, uy, uz, bx, by, bz, inv_len; int parent, a_slot, b_slot; };
struct JitPair { int i, j; float nrs; bool hyd, hb; };            // slots i < j; nrs = -(R_i + R_j)

struct JitDesc {
    int N = 0, T = 0, D = 0;
    std::vector<float> ref;            // [N][3] relative to the pivot
    std::vector<int> map;              // [N] map index
    std::vector<int> frag_of;          // [N]
    std::vector<int> frag_end;         // [T+1]
    std::vector<JitTors> tors;
    std::vector<JitPair> pairs;
};

int build_desc(const dock_params *p, const dock_grid *g, const dock_ligand *L, JitDesc &d)
{
    TppLigand tl;
    std::vector<uint4> overflow;
    if (dock_compile_tpp(p, g, L, tl, overflow) != DOCK_OK) return DOCK_EINVAL;   // validation + slot tables
    const int N = L->N, T = L->T;
    d.N = N; d.T = T; d.D = (N + 1) / 2;
    std::vector<int> atom_of(N), slot_of(N);
    for (int i = 0; i < N; ++i) atom_of[i] = i;
    std::stable_sort(atom_of.begin(), atom_of.end(), [&](int a, int b) { return L->atom_fragment[a] < L->atom_fragment[b]; });
    for (int s = 0; s < N; ++s) slot_of[atom_of[s]] = s;
    d.ref.resize(3 * N); d.map.resize(N); d.frag_of.resize(N);
    for (int s = 0; s < N; ++s) {
        d.ref[3 * s] = tl.atom_ref[s].x; d.ref[3 * s + 1] = tl.atom_ref[s].y; d.ref[3 * s + 2] = tl.atom_ref[s].z;
        d.map[s] = g->type_to_map[L->type[atom_of[s]]];
        d.frag_of[s] = L->atom_fragment[atom_of[s]];
    }
    d.frag_end.resize(T + 1);
    for (int f = 0; f <= T; ++f) d.frag_end[f] = tl.frag_end[f];
    d.tors.resize(T);
    for (int k = 0; k < T; ++k) {
        JitTors &t = d.tors[k];
        t.ux = tl.tors_axis[k].x; t.uy = tl.tors_axis[k].y; t.uz = tl.tors_axis[k].z;
        std::memcpy(&t.parent, &tl.tors_axis[k].w, 4);
        t.bx = tl.tors_pt[k].x; t.by = tl.tors_pt[k].y; t.bz = tl.tors_pt[k].z; t.inv_len = tl.tors_pt[k].w;
        t.a_slot = tl.tors_a[k]; t.b_slot = tl.tors_b[k];
    }
    d.pairs.clear();
    for (int k = 0; k < L->P; ++k) {
        const int ai = L->pairs[2 * k], aj = L->pairs[2 * k + 1];
        int si = slot_of[ai], sj = slot_of[aj];
        if (si > sj) std::swap(si, sj);
        const int ti = L->type[ai], tj = L->type[aj];
        JitPair q;
        q.i = si; q.j = sj;
        q.nrs = -(p->radius[ti] + p->radius[tj]);
        q.hyd = p->hydrophobic[ti] && p->hydrophobic[tj] && p->w[3] != 0.f;
        q.hb = ((p->donor[ti] && p->acceptor[tj]) || (p->donor[tj] && p->acceptor[ti])) && p->w[4] != 0.f;
        d.pairs.push_back(q);
    }
    return DOCK_OK;
}

// ---- source text ------------------------------------------------------------------------------------
struct Src {
    std::string s;
    void operator()(const char *fmt, ...) __attribute__((format(printf, 2, 3)))
    {
        char buf[2048];
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(buf, sizeof buf, fmt, ap);
        va_end(ap);
        s += buf;
        s += '\n';
    }
};

std::string F(float v)                                  // exact fp32 literal
{
    char b[64];
    if (std::isfinite(v)) snprintf(b, sizeof b, "%af", (double)v);
    else {
        unsigned u;
        std::memcpy(&u, &v, 4);
        snprintf(b, sizeof b, "__uint_as_float(0x%08xu)", u);
    }
    return b;
}
#define FS(v) F(v).c_str()

const char *k_prelude = R"SRC(
typedef unsigned long long f32x2;
struct __align__(32) Cell8 { float4 lo, hi; };
__device__ __forceinline__ f32x2 pk2(float lo, float hi) { f32x2 r; asm("mov.b64 %0, {%1,%2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ f32x2 bc2(float v) { return pk2(v, v); }
__device__ __forceinline__ void up2(f32x2 v, float &lo, float &hi) { asm("mov.b64 {%0,%1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ float sum2(f32x2 v) { float a, b; up2(v, a, b); return a + b; }
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) { f32x2 d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d; }
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) { f32x2 d; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) { f32x2 d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ f32x2 sub2(f32x2 a, f32x2 b) { f32x2 d; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ float ex2(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float rsq(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ void ldg_cell(const Cell8 *p, float4 &lo, float4 &hi)
{
    unsigned long long a, b, c, d;
    // volatile: the gathers of the NEXT loop iteration must stay ahead of the interpolation of the current one (pin4)
    asm volatile("ld.global.nc.v4.b64 {%0,%1,%2,%3}, [%4];" : "=l"(a), "=l"(b), "=l"(c), "=l"(d) : "l"(p));
    lo.x = __uint_as_float((unsigned)a); lo.y = __uint_as_float((unsigned)(a >> 32));
    lo.z = __uint_as_float((unsigned)b); lo.w = __uint_as_float((unsigned)(b >> 32));
    hi.x = __uint_as_float((unsigned)c); hi.y = __uint_as_float((unsigned)(c >> 32));
    hi.z = __uint_as_float((unsigned)d); hi.w = __uint_as_float((unsigned)(d >> 32));
}
// an empty volatile statement that "rewrites" v: volatile statements keep their order, so everything that uses v afterwards
// stays behind the volatile loads issued before it (without it the compiler sinks the next iteration's gathers below the
// interpolation of the current one and their latency is exposed: 16 % of all stall samples, profiles/r2b.md)
__device__ __forceinline__ void pin4(float4 &v) { asm volatile("" : "+f"(v.x), "+f"(v.y), "+f"(v.z), "+f"(v.w)); }
// quad image (JIT_QUAD): entry (ix,iy,iz) = the four (x,y) corners of the cell in plane iz; planes iz and iz+1 are adjacent
__device__ __forceinline__ void ldg_quad(const float4 *p, float4 &lo, float4 &hi)
{
    asm volatile("ld.global.nc.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(lo.x), "=f"(lo.y), "=f"(lo.z), "=f"(lo.w) : "l"(p));
    asm volatile("ld.global.nc.v4.f32 {%0,%1,%2,%3}, [%4+16];" : "=f"(hi.x), "=f"(hi.y), "=f"(hi.z), "=f"(hi.w) : "l"(p));
}
// the same gather with an L2 cache hint (policy from createpolicy: evict_last keeps the map image in L2 against the
// streaming poses and outputs)
__device__ __forceinline__ void ldg_cell_hint(const Cell8 *p, float4 &lo, float4 &hi, unsigned long long pol)
{
    unsigned long long a, b, c, d;
    asm volatile("ld.global.nc.L2::cache_hint.v4.b64 {%0,%1,%2,%3}, [%4], %5;" : "=l"(a), "=l"(b), "=l"(c), "=l"(d) : "l"(p), "l"(pol));
    lo.x = __uint_as_float((unsigned)a); lo.y = __uint_as_float((unsigned)(a >> 32));
    lo.z = __uint_as_float((unsigned)b); lo.w = __uint_as_float((unsigned)(b >> 32));
    hi.x = __uint_as_float((unsigned)c); hi.y = __uint_as_float((unsigned)(c >> 32));
    hi.z = __uint_as_float((unsigned)d); hi.w = __uint_as_float((unsigned)(d >> 32));
}
// volatile: the loads stay where the generator put them (one group ahead of their use) and are not forwarded from
// the phase-1 stores, which would pin every coordinate in a register
__device__ __forceinline__ float4 lds4(const float4 *p)
{
    float4 v; const unsigned a = (unsigned)__cvta_generic_to_shared(p);
    asm volatile("ld.volatile.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a));
    return v;
}
__device__ __forceinline__ float2 lds2(const float2 *p)
{
    float2 v; const unsigned a = (unsigned)__cvta_generic_to_shared(p);
    asm volatile("ld.volatile.shared.v2.f32 {%0,%1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(a));
    return v;
}
// sin / cos, |x| < 1.2e4: Cody-Waite reduction + minimax polynomials (same as mathx.cuh)
__device__ __forceinline__ void sincos_cw(float x, float &s, float &c)
{
    const float kf = rintf(x * 0.63661975f);
    float r = fmaf(kf, -1.5703125f, x);
    r = fmaf(kf, -4.837512969970703e-4f, r);
    r = fmaf(kf, -7.549533620476723e-8f, r);
    r = fmaf(kf, -2.5633440682570896e-12f, r);
    const int q = (int)kf;
    const float z = r * r;
    float ps = fmaf(z, -1.9515295891e-4f, 8.3321608736e-3f);
    ps = fmaf(ps, z, -1.6666654611e-1f);
    ps = fmaf(ps * z, r, r);
    float pc = fmaf(z, 2.443315711809948e-5f, -1.388731625493765e-3f);
    pc = fmaf(pc, z, 4.166664568298827e-2f);
    pc = fmaf(pc * z, z, fmaf(-0.5f, z, 1.0f));
    const float ss = (q & 1) ? pc : ps;
    const float cc = (q & 1) ? ps : pc;
    s = (q & 2) ? -ss : ss;
    c = ((q + 1) & 2) ? -cc : cc;
}
struct CellRef { int idx; float px, py, pz, ox, oy, oz; };
__device__ __forceinline__ CellRef locate_cell(const JitArgs &G, float x, float y, float z)
{
    const float ux = fmaf(x, G.inv_h_lo, x * G.inv_h);
    const float uy = fmaf(y, G.inv_h_lo, y * G.inv_h);
    const float uz = fmaf(z, G.inv_h_lo, z * G.inv_h);
    const float cx = fminf(fmaxf(ux, G.lo_x), G.hi_x);
    const float cy = fminf(fmaxf(uy, G.lo_y), G.hi_y);
    const float cz = fminf(fmaxf(uz, G.lo_z), G.hi_z);
    CellRef c;
    c.ox = ux - cx; c.oy = uy - cy; c.oz = uz - cz;
    const float fx = fminf(floorf(cx), G.hi_x - 1.0f);
    const float fy = fminf(floorf(cy), G.hi_y - 1.0f);
    const float fz = fminf(floorf(cz), G.hi_z - 1.0f);
    c.px = cx - fx; c.py = cy - fy; c.pz = cz - fz;
    const int ix = (int)fx + G.icx, iy = (int)fy + G.icy, iz = (int)fz + G.icz;
    c.idx = JIT_QUAD ? (iy * G.nx + ix) * G.nz + iz : (iz * G.ny + iy) * G.nx + ix;
    return c;
}
// the index part of locate_cell alone, and an L2 prefetch of the cell
__device__ __forceinline__ int cell_index(const JitArgs &G, float x, float y, float z)
{
    const float ux = fmaf(x, G.inv_h_lo, x * G.inv_h), uy = fmaf(y, G.inv_h_lo, y * G.inv_h), uz = fmaf(z, G.inv_h_lo, z * G.inv_h);
    const float fx = fminf(floorf(fminf(fmaxf(ux, G.lo_x), G.hi_x)), G.hi_x - 1.0f);
    const float fy = fminf(floorf(fminf(fmaxf(uy, G.lo_y), G.hi_y)), G.hi_y - 1.0f);
    const float fz = fminf(floorf(fminf(fmaxf(uz, G.lo_z), G.hi_z)), G.hi_z - 1.0f);
    const int ix = (int)fx + G.icx, iy = (int)fy + G.icy, iz = (int)fz + G.icz;
    return JIT_QUAD ? (iy * G.nx + ix) * G.nz + iz : (iz * G.ny + iy) * G.nx + ix;
}
__device__ __forceinline__ void prefetch_l2(const void *p) { asm volatile("prefetch.global.L2 [%0];" :: "l"(p)); }
// eq. 2 + eq. 3 + wall (reading S7).  Same interpolant as mathx.cuh::trilinear, evaluated z first, then y, then x so that
// the four (x,y) corners of a plane run two per fp32x2 instruction: 8 packed + 6 scalar instructions instead of 22.
__device__ __forceinline__ float trilinear(const JitArgs &G, const CellRef &c, const float4 q0, const float4 q1,
                                           float &e_wall, float &gx, float &gy, float &gz)
{
    const f32x2 lo0 = pk2(q0.x, q0.y), hi0 = pk2(q0.z, q0.w);             // plane iz: (x0,x1) at y0, (x0,x1) at y1
    const f32x2 dzl = sub2(pk2(q1.x, q1.y), lo0), dzh = sub2(pk2(q1.z, q1.w), hi0);
    const f32x2 pz2 = bc2(c.pz), py2 = bc2(c.py);
    const f32x2 cl = fma2(pz2, dzl, lo0), ch = fma2(pz2, dzh, hi0);        // interpolated along z
    const f32x2 dy = sub2(ch, cl);
    const f32x2 cy = fma2(py2, dy, cl);                                    // ... along y: (value at x0, value at x1)
    const f32x2 dzy = fma2(py2, sub2(dzh, dzl), dzl);                      // d/dz interpolated along y
    float c0, c1, dy0, dy1, dz0, dz1;
    up2(cy, c0, c1); up2(dy, dy0, dy1); up2(dzy, dz0, dz1);
    const float ex = c1 - c0;
    const float e = fmaf(c.px, ex, c0);                                    // eq. 2
    float ggx = ex * G.inv_h;                                              // eq. 3
    float ggy = fmaf(c.px, dy1 - dy0, dy0) * G.inv_h;
    float ggz = fmaf(c.px, dz1 - dz0, dz0) * G.inv_h;
    if (c.ox != 0.0f) ggx = 0.0f;
    if (c.oy != 0.0f) ggy = 0.0f;
    if (c.oz != 0.0f) ggz = 0.0f;
    gx = fmaf(G.kw_g, c.ox, ggx);
    gy = fmaf(G.kw_g, c.oy, ggy);
    gz = fmaf(G.kw_g, c.oz, ggz);
    e_wall = fmaf(G.kw_e, fmaf(c.ox, c.ox, fmaf(c.oy, c.oy, c.oz * c.oz)), e_wall);
    return e;
}
)SRC";

// float4 units of shared memory per warp: coordinates (D x 48) + region 2 = max(frames 12 T floats, grid forces 6 D floats) per lane
int jit_warp_float4(int N, int T, bool want_grad)
{
    const int D = (N + 1) / 2;
    const int r2 = std::max(want_grad ? 6 * D : 0, 13 * T);        // floats per lane (frames 12 T + staged torsion angles T)
    return D * 48 + (r2 * 32 + 3) / 4;
}

// One chain = two pairs in the two lanes of fp32x2 registers (or one pair, scalar).  Lane l pairs atom ta[l] of the
// tile duo with partner atom pa[l].
enum { CH_SCALAR = 0, CH_BCAST = 1, CH_DIAG = 2, CH_GEN = 3 };
struct Chain {
    int kind;
    int tile;              // tile duo (packed kinds); lanes = its two atoms in order
    int ta[2], pa[2];      // atoms of the pair in lane l (scalar: lane 0 only)
    float nrs[2];
    bool hyd[2], hb[2];
    bool inr[2];           // the pair can never reach the cutoff (upper bound of its distance over all torsion angles)
};

struct Gen {
    const JitDesc &d;
    const JitOpts &o;
    Src S;
    std::vector<int> duo_of, half_of;      // atom -> duo, lane
    std::vector<int> mem;                  // [D][2] duo -> atoms (-1 = padding)
    std::vector<int> pid;                  // [N][N] pair index or -1
    Gen(const JitDesc &d_, const JitOpts &o_) : d(d_), o(o_) {}
    // the pair-term constants (DevParams) are baked in as literals: immediates instead of constant-bank loads
    float cutoff = 0.f;
    std::string k_cutoff2, k_lw1, k_lw2b, k_q, k_m3q, k_c4, k_sigma, k_eA, k_eB, k_whp, k_whbp;
    void set_params(const dock_params *p, const DevParams &P)
    {
        cutoff = P.cutoff;
        k_cutoff2 = F(P.cutoff2); k_lw1 = F(P.lw1); k_lw2b = F(P.lw2 - 3.2460638420001677f); k_q = F(P.q); k_m3q = F(P.m3q);
        k_c4 = F(P.c4); k_sigma = F(P.sigma); k_eA = F(P.eA); k_eB = F(P.eB);
        k_whp = F(-P.sigma * p->w[3]);
        k_whbp = F((float)(-(double)P.sigma * (double)p->w[4] / 0.7));
    }

    // ---- duos: which two atoms share a register pair ---------------------------------------------------
    int listed(int a, int b) const { return (a >= 0 && b >= 0 && a != b) ? pid[(size_t)a * d.N + b] : -1; }
    // Upper bound of |x_a - x_b| over all poses: both axis atoms of a torsion keep their distance to every atom of the
    // two fragments the torsion joins, so the triangle inequality along the fragment path bounds the distance.
    float refdist(int a, int b) const
    {
        const float dx = d.ref[3 * a] - d.ref[3 * b], dy = d.ref[3 * a + 1] - d.ref[3 * b + 1], dz = d.ref[3 * a + 2] - d.ref[3 * b + 2];
        return std::sqrt(dx * dx + dy * dy + dz * dz);
    }
    float max_dist(int a, int b) const
    {
        int fa = d.frag_of[a], fb = d.frag_of[b];
        if (fa == fb) return refdist(a, b);
        std::vector<int> up_a, up_b;                        // torsions from each fragment towards the root
        auto parent = [&](int f) { return d.tors[f - 1].parent; };
        std::vector<int> anc_a;
        for (int f = fa; ; f = parent(f)) { anc_a.push_back(f); if (f == 0) break; }
        int lca = fb;
        std::vector<int> path_b;
        for (;; lca = parent(lca)) {
            if (std::find(anc_a.begin(), anc_a.end(), lca) != anc_a.end()) break;
            path_b.push_back(lca - 1);                      // torsion joining lca to its parent
        }
        std::vector<int> path;                              // torsions in order from a's fragment to b's
        for (int f = fa; f != lca; f = parent(f)) path.push_back(f - 1);
        for (int k = (int)path_b.size() - 1; k >= 0; --k) path.push_back(path_b[k]);
        float best[2] = {0.f, 0.f};
        for (size_t l = 0; l < path.size(); ++l) {
            const int q[2] = {d.tors[path[l]].a_slot, d.tors[path[l]].b_slot};
            float nb[2];
            for (int c = 0; c < 2; ++c) {
                if (l == 0) nb[c] = refdist(a, q[c]);
                else {
                    const int pq[2] = {d.tors[path[l - 1]].a_slot, d.tors[path[l - 1]].b_slot};
                    nb[c] = std::min(best[0] + refdist(pq[0], q[c]), best[1] + refdist(pq[1], q[c]));
                }
            }
            best[0] = nb[0]; best[1] = nb[1];
        }
        const int lq[2] = {d.tors[path.back()].a_slot, d.tors[path.back()].b_slot};
        return std::min(best[0] + refdist(lq[0], b), best[1] + refdist(lq[1], b));
    }
    // chains needed for the pairs between duos A and B (or inside A when A == B)
    int block_cost(const int *ma, const int *mb, bool same) const
    {
        if (same) return listed(ma[0], ma[1]) >= 0 ? 1 : 0;
        int n = 0;
        for (int i = 0; i < 2; ++i) for (int j = 0; j < 2; ++j) n += listed(ma[i], mb[j]) >= 0;
        return (n + 1) / 2;
    }
    int total_cost() const
    {
        int c = 0;
        for (int A = 0; A < d.D; ++A)
            for (int B = A; B < d.D; ++B) c += block_cost(&mem[2 * A], &mem[2 * B], A == B);
        return c;
    }
    void choose_duos()
    {
        const int N = d.N, D = d.D;
        pid.assign((size_t)N * N, -1);
        for (size_t k = 0; k < d.pairs.size(); ++k) {
            pid[(size_t)d.pairs[k].i * N + d.pairs[k].j] = (int)k;
            pid[(size_t)d.pairs[k].j * N + d.pairs[k].i] = (int)k;
        }
        mem.assign(2 * D, -1);
        for (int a = 0; a < N; ++a) mem[a] = a;                     // start: consecutive atoms (fragment order)
        // local search: exchange one atom between two duos while the number of chains goes down (deterministic)
        int best = total_cost();
        for (bool improved = true; improved;) {
            improved = false;
            for (int A = 0; A < D; ++A)
                for (int B = A + 1; B < D; ++B)
                    for (int i = 0; i < 2; ++i)
                        for (int j = 0; j < 2; ++j) {
                            if (mem[2 * A + i] < 0 && mem[2 * B + j] < 0) continue;
                            std::swap(mem[2 * A + i], mem[2 * B + j]);
                            const int c = total_cost();
                            if (c < best) { best = c; improved = true; }
                            else std::swap(mem[2 * A + i], mem[2 * B + j]);
                        }
        }
        for (int dd = 0; dd < D; ++dd)                              // padding goes to lane 1
            if (mem[2 * dd] < 0) std::swap(mem[2 * dd], mem[2 * dd + 1]);
        duo_of.assign(N, 0); half_of.assign(N, 0);
        for (int dd = 0; dd < D; ++dd)
            for (int h = 0; h < 2; ++h)
                if (mem[2 * dd + h] >= 0) { duo_of[mem[2 * dd + h]] = dd; half_of[mem[2 * dd + h]] = h; }
    }

    // ---- coordinates: loaded per group from shared memory (volatile: see lds4) ---------------------------
    std::vector<int> last_load;            // duo -> group tag of its most recent load (-100 = never)
    std::string cvar(int duo, int tag) { char b[48]; snprintf(b, sizeof b, "cq%d_%d", tag, duo); return b; }
    std::string wvar(int duo, int tag) { char b[48]; snprintf(b, sizeof b, "wq%d_%d", tag, duo); return b; }
    // makes duo's coordinates available to code emitted for group g; returns the tag of the variables to use
    int need_duo(int duo, int g)
    {
        if (last_load[duo] >= g - o.reuse) return last_load[duo];
        last_load[duo] = g;
        S("    const float4 %s = lds4(xyq + %d); const float2 %s = lds2(zq + %d);", cvar(duo, g).c_str(), duo * 32, wvar(duo, g).c_str(), duo * 32);
        return g;
    }
    int tag_of(int duo) const { return last_load[duo]; }
    std::string sx(int a) { return cvar(duo_of[a], tag_of(duo_of[a])) + (half_of[a] ? ".y" : ".x"); }
    std::string sy(int a) { return cvar(duo_of[a], tag_of(duo_of[a])) + (half_of[a] ? ".w" : ".z"); }
    std::string sz(int a) { return wvar(duo_of[a], tag_of(duo_of[a])) + (half_of[a] ? ".y" : ".x"); }
    std::string px(int duo) { const std::string c = cvar(duo, tag_of(duo)); return "pk2(" + c + ".x, " + c + ".y)"; }
    std::string py(int duo) { const std::string c = cvar(duo, tag_of(duo)); return "pk2(" + c + ".z, " + c + ".w)"; }
    std::string pz(int duo) { const std::string c = wvar(duo, tag_of(duo)); return "pk2(" + c + ".x, " + c + ".y)"; }

    // ---- A2 as loops over fragments and atoms (compact code; tables in the constant bank).  Frames of fragments
    // 0..T-1 live in shared memory (region 2, which holds the grid forces later) so that a child can fetch its parent's
    void kinematics()
    {
        const int T = d.T;
        S("    // ---- phase 1: A2 ----");
        S("    {");
        S("    float2 *const fr = reinterpret_cast<float2 *>(reg2) + lane;     // [T][6], stride 32");
        S("    float m00, m01, m02, m10, m11, m12, m20, m21, m22, c0 = 0.0f, c1 = 0.0f, c2 = 0.0f;");
        S("    {");
        S("        float w = POSE(3), x = POSE(4), y = POSE(5), z = POSE(6);");
        S("        const float n2 = fmaf(w, w, fmaf(x, x, fmaf(y, y, z * z)));");
        S("        if (n2 > 0.0f) { const float inv = 1.0f / sqrtf(n2); w *= inv; x *= inv; y *= inv; z *= inv; } else { w = 1.0f; x = y = z = 0.0f; }");
        S("        const float x2 = x + x, y2 = y + y, z2 = z + z;");
        S("        m00 = 1.0f - fmaf(y2, y, z2 * z); m01 = fmaf(x2, y, -w * z2); m02 = fmaf(x2, z, w * y2);");
        S("        m10 = fmaf(x2, y, w * z2); m11 = 1.0f - fmaf(x2, x, z2 * z); m12 = fmaf(y2, z, -w * x2);");
        S("        m20 = fmaf(x2, z, -w * y2); m21 = fmaf(y2, z, w * x2); m22 = 1.0f - fmaf(x2, x, y2 * y);");
        S("    }");
        S("    float *const xyf = reinterpret_cast<float *>(xyq), *const zf = reinterpret_cast<float *>(zq);");
        if (T > 0) {                                          // all torsion angles in one burst (one exposed load latency)
            S("    float *const thf = reinterpret_cast<float *>(reg2) + %d + lane;", 12 * T * 32);
            S("    #pragma unroll");
            S("    for (int k = 0; k < %d; ++k) thf[k * 32] = POSE(7 + k);", T);
        }
        S("    int s = 0;");
        S("    #pragma unroll 1");
        S("    for (int f = 0; f <= %d; ++f) {", T);
        if (T > 0) {
            S("        if (f > 0) {");
            S("            const JitF3I u = jit_axis[f - 1]; const float4 b = jit_pt[f - 1];");
            S("            const int pf = u.w;");
            S("            float sn, cs; sincos_cw(thf[(f - 1) * 32], sn, cs);");
            S("            const float2 p0 = fr[(6 * pf) * 32], p1 = fr[(6 * pf + 1) * 32], p2 = fr[(6 * pf + 2) * 32];");
            S("            const float2 p3 = fr[(6 * pf + 3) * 32], p4 = fr[(6 * pf + 4) * 32], p5 = fr[(6 * pf + 5) * 32];");
            S("            const float omc = 1.0f - cs;");
            S("            const float ox = omc * u.x, oy = omc * u.y, oz = omc * u.z;");
            S("            const float sx = sn * u.x, sy = sn * u.y, sz = sn * u.z;");
            S("            const float r00 = fmaf(ox, u.x, cs), r01 = fmaf(ox, u.y, -sz), r02 = fmaf(ox, u.z, sy);");
            S("            const float r10 = fmaf(ox, u.y, sz), r11 = fmaf(oy, u.y, cs), r12 = fmaf(oy, u.z, -sx);");
            S("            const float r20 = fmaf(ox, u.z, -sy), r21 = fmaf(oy, u.z, sx), r22 = fmaf(oz, u.z, cs);");
            S("            const float v0 = b.x - fmaf(r00, b.x, fmaf(r01, b.y, r02 * b.z));");
            S("            const float v1 = b.y - fmaf(r10, b.x, fmaf(r11, b.y, r12 * b.z));");
            S("            const float v2 = b.z - fmaf(r20, b.x, fmaf(r21, b.y, r22 * b.z));");
            S("            c0 = fmaf(p0.x, v0, fmaf(p0.y, v1, fmaf(p1.x, v2, p4.y)));");
            S("            c1 = fmaf(p1.y, v0, fmaf(p2.x, v1, fmaf(p2.y, v2, p5.x)));");
            S("            c2 = fmaf(p3.x, v0, fmaf(p3.y, v1, fmaf(p4.x, v2, p5.y)));");
            S("            m00 = fmaf(p0.x, r00, fmaf(p0.y, r10, p1.x * r20)); m01 = fmaf(p0.x, r01, fmaf(p0.y, r11, p1.x * r21)); m02 = fmaf(p0.x, r02, fmaf(p0.y, r12, p1.x * r22));");
            S("            m10 = fmaf(p1.y, r00, fmaf(p2.x, r10, p2.y * r20)); m11 = fmaf(p1.y, r01, fmaf(p2.x, r11, p2.y * r21)); m12 = fmaf(p1.y, r02, fmaf(p2.x, r12, p2.y * r22));");
            S("            m20 = fmaf(p3.x, r00, fmaf(p3.y, r10, p4.x * r20)); m21 = fmaf(p3.x, r01, fmaf(p3.y, r11, p4.x * r21)); m22 = fmaf(p3.x, r02, fmaf(p3.y, r12, p4.x * r22));");
            S("        }");
            S("        if (f < %d) {", T);
            S("            fr[(6 * f) * 32] = make_float2(m00, m01); fr[(6 * f + 1) * 32] = make_float2(m02, m10); fr[(6 * f + 2) * 32] = make_float2(m11, m12);");
            S("            fr[(6 * f + 3) * 32] = make_float2(m20, m21); fr[(6 * f + 4) * 32] = make_float2(m22, c0); fr[(6 * f + 5) * 32] = make_float2(c1, c2);");
            S("        }");
        }
        S("        const int s_end = jit_frag_end[f];");
        S("        #pragma unroll %d", o.atom_unroll);
        S("        for (; s < s_end; ++s) {");
        S("            const JitF3I r = jit_ref[s];");
        S("            const int sl = r.w & 255, dd = sl >> 1, h = sl & 1;     // duo and lane of this atom (bits 8..: its map)");
        S("            const float ax = fmaf(m00, r.x, fmaf(m01, r.y, fmaf(m02, r.z, c0)));");
        S("            const float ay = fmaf(m10, r.x, fmaf(m11, r.y, fmaf(m12, r.z, c1)));");
        S("            const float az = fmaf(m20, r.x, fmaf(m21, r.y, fmaf(m22, r.z, c2)));");
        S("            xyf[dd * 128 + h] = ax; xyf[dd * 128 + 2 + h] = ay; zf[dd * 64 + h] = az;");
        if (o.prefetch)                                       // the atom's map cell on its way into L2 while the rest of phase 1 runs
            S("            prefetch_l2(maps + ((long long)(r.w >> 8) * a.map_stride + cell_index(a, ax + tx, ay + ty, az + tz)));");
        S("        }");
        S("    }");
        if (d.N & 1) S("    xyf[%d] = 0.0f; xyf[%d] = 0.0f; zf[%d] = 0.0f;", (d.D - 1) * 128 + 1, (d.D - 1) * 128 + 3, (d.D - 1) * 64 + 1);
        S("    }");
    }

    std::string tables()
    {
        std::string t;
        char b[256];
        t += "__constant__ int jit_maps[" + std::to_string(2 * d.D) + "] = {";
        for (int i = 0; i < 2 * d.D; ++i) t += std::to_string(mem[i] >= 0 ? d.map[mem[i]] : 0) + (i + 1 < 2 * d.D ? ", " : "};\n");
        t += "__constant__ int jit_frag_end[" + std::to_string(d.T + 1) + "] = {";
        for (int f = 0; f <= d.T; ++f) t += std::to_string(d.frag_end[f]) + (f < d.T ? ", " : "};\n");
        t += "struct __align__(16) JitF3I { float x, y, z; int w; };\n__constant__ JitF3I jit_ref[" + std::to_string(d.N) + "] = {\n";
        for (int s = 0; s < d.N; ++s) {
            snprintf(b, sizeof b, "    {%s, %s, %s, %d}%s\n", FS(d.ref[3 * s]), FS(d.ref[3 * s + 1]), FS(d.ref[3 * s + 2]),
                     (2 * duo_of[s] + half_of[s]) | (d.map[s] << 8), s + 1 < d.N ? "," : "};");
            t += b;
        }
        if (d.T > 0) {
            t += "__constant__ JitF3I jit_axis[" + std::to_string(d.T) + "] = {\n";
            for (int k = 0; k < d.T; ++k) {
                snprintf(b, sizeof b, "    {%s, %s, %s, %d}%s\n", FS(d.tors[k].ux), FS(d.tors[k].uy), FS(d.tors[k].uz), d.tors[k].parent, k + 1 < d.T ? "," : "};");
                t += b;
            }
            t += "__constant__ float4 jit_pt[" + std::to_string(d.T) + "] = {\n";
            for (int k = 0; k < d.T; ++k) {
                snprintf(b, sizeof b, "    {%s, %s, %s, 0.0f}%s\n", FS(d.tors[k].bx), FS(d.tors[k].by), FS(d.tors[k].bz), k + 1 < d.T ? "," : "};");
                t += b;
            }
        }
        return t;
    }

    // ---- A3: map lookups as a LOOP over the duos (compact code: the i-cache holds ~8 k instructions, profiles/r2b.md);
    // the sigma-scaled grid forces go to shared memory and seed the force registers of the pair phase
    void grid_loop()
    {
        // Two register sets (A, B) of U duos each, ping-pong: while the cells of one set are interpolated the gathers of the
        // other are in flight, with no register copies (a copy of a loaded register waits for the load) and no branch
        // around the requests (ptxas hoists the interpolation above a conditional request).  Indices past the last full
        // duo are clamped and their results masked.
        const int U = o.grid_unroll;
        const int D2 = d.N / 2;                              // full duos
        const int NS = o.grid_sets;                          // register sets: NS - 1 of them are in flight
        const int n_it = (D2 + NS * U - 1) / (NS * U);
        const bool ragged = D2 % (NS * U) != 0;
        S("    // ---- phase 2a: A3 (map lookups), %d x %d atoms per iteration ----", NS, 2 * U);
        S("    float e_grid = 0.0f, e_wall = 0.0f;");
        auto issue = [&](char set, const std::string &dd, int u) {           // locate + gather of duo dd into the set's registers
            S("        { const int di = min(%s, %d); const float4 c = xyq[di * 32]; const float2 w = zq[di * 32];", dd.c_str(), std::max(D2 - 1, 0));
            S("          r%c%da = locate_cell(a, c.x + tx, c.z + ty, w.x + tz); r%c%db = locate_cell(a, c.y + tx, c.w + ty, w.y + tz);", set, u, set, u);
            S("          LDG_CELL(maps + ((long long)jit_maps[2 * di] * a.map_stride + r%c%da.idx), p%c%da0, p%c%da1);", set, u, set, u, set, u);
            S("          LDG_CELL(maps + ((long long)jit_maps[2 * di + 1] * a.map_stride + r%c%db.idx), p%c%db0, p%c%db1); }", set, u, set, u, set, u);
        };
        auto consume = [&](char set, const std::string &dd, int u) {
            S("        { float g0x, g0y, g0z, g1x, g1y, g1z, ew = 0.0f;");
            S("          const float e01 = trilinear(a, r%c%da, p%c%da0, p%c%da1, ew, g0x, g0y, g0z) + trilinear(a, r%c%db, p%c%db0, p%c%db1, ew, g1x, g1y, g1z);", set, u, set, u, set, u, set, u, set, u, set, u);
            if (ragged) {
                S("          const int dd = %s; const bool live = dd < %d;", dd.c_str(), D2);
                S("          e_grid += live ? e01 : 0.0f; e_wall += live ? ew : 0.0f;");
                if (o.want_grad) {
                    S("          if (live) { gq4[dd * 32] = make_float4(K_sigma * g0x, K_sigma * g1x, K_sigma * g0y, K_sigma * g1y);");
                    S("                      gq2[dd * 32] = make_float2(K_sigma * g0z, K_sigma * g1z); }");
                }
            } else {
                S("          const int dd = %s;", dd.c_str());
                S("          e_grid += e01; e_wall += ew;");
                if (o.want_grad) {
                    S("          gq4[dd * 32] = make_float4(K_sigma * g0x, K_sigma * g1x, K_sigma * g0y, K_sigma * g1y);");
                    S("          gq2[dd * 32] = make_float2(K_sigma * g0z, K_sigma * g1z);");
                }
            }
            S("        }");
        };
        if (D2 > 0) {
            S("    {");
            for (int j = 0; j < NS; ++j)
                for (int u = 0; u < U; ++u) {
                    const char c = (char)('A' + j);
                    S("    CellRef r%c%da, r%c%db; float4 p%c%da0, p%c%da1, p%c%db0, p%c%db1;", c, u, c, u, c, u, c, u, c, u, c, u);
                }
            for (int j = 0; j + 1 < NS; ++j)
                for (int u = 0; u < U; ++u) issue((char)('A' + j), std::to_string(j * U + u), u);
            S("    #pragma unroll 1");
            S("    for (int it = 0; it < %d; ++it) {", n_it);
            S("        const int base = it * %d;", NS * U);
            for (int j = 0; j < NS; ++j) {
                const int jn = (j + NS - 1) % NS;          // the set consumed longest ago is refilled, NS - 1 sets ahead
                for (int u = 0; u < U; ++u) issue((char)('A' + jn), "base + " + std::to_string((j + NS - 1) * U + u), u);
                for (int u = 0; u < U; ++u) consume((char)('A' + j), "base + " + std::to_string(j * U + u), u);
            }
            S("    }");
            S("    }");
        }
        if (d.N & 1) {                                      // the single atom of an odd ligand
            const int dd = d.D - 1;
            S("    {");
            S("        const float4 c = xyq[%d]; const float2 w = zq[%d];", dd * 32, dd * 32);
            S("        const CellRef r0 = locate_cell(a, c.x + tx, c.z + ty, w.x + tz);");
            S("        float4 p0, p1; LDG_CELL(maps + (%dLL * a.map_stride + r0.idx), p0, p1);", d.map[mem[2 * dd]]);
            S("        float g0x, g0y, g0z; e_grid += trilinear(a, r0, p0, p1, e_wall, g0x, g0y, g0z);");
            if (o.want_grad) {
                S("        gq4[%d] = make_float4(K_sigma * g0x, 0.0f, K_sigma * g0y, 0.0f);", dd * 32);
                S("        gq2[%d] = make_float2(K_sigma * g0z, 0.0f);", dd * 32);
            }
            S("    }");
        }
    }

    std::vector<Chain> chains;
    void add_chain(int kind, int tile, int t0, int p0, int t1, int p1)
    {
        Chain c;
        c.kind = kind; c.tile = tile;
        c.ta[0] = t0; c.pa[0] = p0; c.ta[1] = t1; c.pa[1] = p1;
        for (int l = 0; l < 2; ++l) {
            const int k = (kind == CH_SCALAR && l == 1) ? -1 : listed(c.ta[l], c.pa[l]);
            c.nrs[l] = k >= 0 ? d.pairs[k].nrs : 0.f;
            c.hyd[l] = k >= 0 && d.pairs[k].hyd;
            c.hb[l] = k >= 0 && d.pairs[k].hb;
            c.inr[l] = k >= 0 && max_dist(c.ta[l], c.pa[l]) < cutoff - 0.05f;
        }
        chains.push_back(c);
    }
    void build_chains()
    {
        for (int A = 0; A < d.D; ++A) {
            const int a0 = mem[2 * A], a1 = mem[2 * A + 1];
            if (listed(a0, a1) >= 0) add_chain(CH_SCALAR, A, a0, a1, -1, -1);
            for (int B = A + 1; B < d.D; ++B) {
                const int b0 = mem[2 * B], b1 = mem[2 * B + 1];
                const bool l00 = listed(a0, b0) >= 0, l01 = listed(a0, b1) >= 0, l10 = listed(a1, b0) >= 0, l11 = listed(a1, b1) >= 0;
                const int n = l00 + l01 + l10 + l11;
                if (n == 0) continue;
                if (n == 4) { add_chain(CH_BCAST, A, a0, b0, a1, b0); add_chain(CH_BCAST, A, a0, b1, a1, b1); }
                else if (n == 3) {
                    if (!l11) { add_chain(CH_BCAST, A, a0, b0, a1, b0); add_chain(CH_SCALAR, A, a0, b1, -1, -1); }
                    else if (!l10) { add_chain(CH_BCAST, A, a0, b1, a1, b1); add_chain(CH_SCALAR, A, a0, b0, -1, -1); }
                    else if (!l01) { add_chain(CH_BCAST, A, a0, b0, a1, b0); add_chain(CH_SCALAR, A, a1, b1, -1, -1); }
                    else { add_chain(CH_BCAST, A, a0, b1, a1, b1); add_chain(CH_SCALAR, A, a1, b0, -1, -1); }
                } else if (n == 2) {
                    if (l00 && l10) add_chain(CH_BCAST, A, a0, b0, a1, b0);
                    else if (l01 && l11) add_chain(CH_BCAST, A, a0, b1, a1, b1);
                    else if (l00 && l01) add_chain(CH_BCAST, B, b0, a0, b1, a0);
                    else if (l10 && l11) add_chain(CH_BCAST, B, b0, a1, b1, a1);
                    else if (l00 && l11) add_chain(CH_DIAG, A, a0, b0, a1, b1);
                    else add_chain(CH_GEN, A, a0, b1, a1, b0);
                } else {
                    if (l00) add_chain(CH_SCALAR, A, a0, b0, -1, -1);
                    else if (l01) add_chain(CH_SCALAR, A, a0, b1, -1, -1);
                    else if (l10) add_chain(CH_SCALAR, A, a1, b0, -1, -1);
                    else add_chain(CH_SCALAR, A, a1, b1, -1, -1);
                }
            }
        }
    }

    // scalar force update of atom b: g_b += sgn * k * (dx, dy, dz)
    void force_scalar(int b, const char *sgn, const char *k, const char *x, const char *y, const char *z)
    {
        S("      gx%d = fmaf(%s%s, %s, gx%d); gy%d = fmaf(%s%s, %s, gy%d); gz%d = fmaf(%s%s, %s, gz%d);", b, sgn, k, x, b, b, sgn, k, y, b, b, sgn, k, z, b);
    }

    void pair_phase()
    {
        build_chains();
        const int K = o.group;
        const int n = (int)chains.size();
        const int n_groups = (n + K - 1) / K;
        last_load.assign(d.D, -100);
        S("    // ---- phase 2b: A4, %d chains for %zu pairs ----", n, d.pairs.size());
        S("    const f32x2 zero2 = bc2(0.0f);");
        S("    f32x2 accA0 = zero2, accB0 = zero2, accR0 = zero2, accA1 = zero2, accB1 = zero2, accR1 = zero2, accH = zero2, accHB = zero2;");
        S("    float sA = 0.0f, sB = 0.0f, sR = 0.0f;");
        S("    const f32x2 WH11 = bc2(K_whp), WH10 = pk2(K_whp, 0.0f), WH01 = pk2(0.0f, K_whp);");
        S("    const f32x2 WB11 = bc2(K_whbp), WB10 = pk2(K_whbp, 0.0f), WB01 = pk2(0.0f, K_whbp);");
        if (o.want_grad)                                    // force registers start from the grid forces
            for (int dd = 0; dd < d.D; ++dd) {
                const int a0 = mem[2 * dd], a1 = mem[2 * dd + 1];
                S("    const float4 gi4_%d = gq4[%d]; const float2 gi2_%d = gq2[%d];", dd, dd * 32, dd, dd * 32);
                S("    float gx%d = gi4_%d.x, gy%d = gi4_%d.z, gz%d = gi2_%d.x;", a0, dd, a0, dd, a0, dd);
                if (a1 >= 0) S("    float gx%d = gi4_%d.y, gy%d = gi4_%d.w, gz%d = gi2_%d.y;", a1, dd, a1, dd, a1, dd);
            }
        auto emit_loads = [&](int g) {
            for (int c = g * K; c < std::min(n, (g + 1) * K); ++c) {
                const Chain &ch = chains[c];
                for (int l = 0; l < (ch.kind == CH_SCALAR ? 1 : 2); ++l) { need_duo(duo_of[ch.ta[l]], g); need_duo(duo_of[ch.pa[l]], g); }
            }
        };
        if (n_groups > 0) emit_loads(0);
        for (int g = 0; g < n_groups; ++g) {
            S("    // group %d", g);
            if (o.sync_every > 0 && g > 0 && g % o.sync_every == 0) S("    __syncthreads();");
            const int c0 = g * K, c1 = std::min(n, (g + 1) * K);
            // stage 1: distances (operands were loaded one group ahead; the next group's loads follow)
            for (int c = c0; c < c1; ++c) {
                const Chain &ch = chains[c];
                if (ch.kind == CH_SCALAR) {
                    S("    const float dx%d = %s - %s, dy%d = %s - %s, dz%d = %s - %s;", c, sx(ch.ta[0]).c_str(), sx(ch.pa[0]).c_str(), c, sy(ch.ta[0]).c_str(), sy(ch.pa[0]).c_str(), c, sz(ch.ta[0]).c_str(), sz(ch.pa[0]).c_str());
                    S("    const float r2%d = fmaf(dz%d, dz%d, fmaf(dy%d, dy%d, fmaf(dx%d, dx%d, 1e-12f)));", c, c, c, c, c, c, c);
                    continue;
                }
                std::string bxs, bys, bzs;
                if (ch.kind == CH_BCAST) { bxs = "bc2(" + sx(ch.pa[0]) + ")"; bys = "bc2(" + sy(ch.pa[0]) + ")"; bzs = "bc2(" + sz(ch.pa[0]) + ")"; }
                else if (ch.kind == CH_DIAG) { const int B = duo_of[ch.pa[0]]; bxs = px(B); bys = py(B); bzs = pz(B); }
                else { bxs = "pk2(" + sx(ch.pa[0]) + ", " + sx(ch.pa[1]) + ")"; bys = "pk2(" + sy(ch.pa[0]) + ", " + sy(ch.pa[1]) + ")"; bzs = "pk2(" + sz(ch.pa[0]) + ", " + sz(ch.pa[1]) + ")"; }
                S("    const f32x2 dx%d = sub2(%s, %s), dy%d = sub2(%s, %s), dz%d = sub2(%s, %s);", c, px(ch.tile).c_str(), bxs.c_str(), c, py(ch.tile).c_str(), bys.c_str(), c, pz(ch.tile).c_str(), bzs.c_str());
                S("    const f32x2 r2%d = fma2(dz%d, dz%d, fma2(dy%d, dy%d, fma2(dx%d, dx%d, bc2(1e-12f))));", c, c, c, c, c, c, c);
            }
            // stage 2: reciprocal square roots
            for (int c = c0; c < c1; ++c) {
                if (chains[c].kind == CH_SCALAR) S("    const float ri%d = rsq(r2%d);", c, c);
                else {
                    S("    float r2l%d, r2h%d; up2(r2%d, r2l%d, r2h%d);", c, c, c, c, c);
                    S("    const f32x2 ri%d = pk2(rsq(r2l%d), rsq(r2h%d));", c, c, c);
                }
            }
            if (g + 1 < n_groups) emit_loads(g + 1);
            // stage 3: surface distance, cutoff, exponent arguments, repulsion
            for (int c = c0; c < c1; ++c) {
                const Chain &ch = chains[c];
                const int k = c & 1;
                if (ch.kind != CH_SCALAR) {
                    if (ch.nrs[0] == ch.nrs[1]) S("    const f32x2 d0%d = fma2(r2%d, ri%d, bc2(%s));", c, c, c, FS(ch.nrs[0]));
                    else S("    const f32x2 d0%d = fma2(r2%d, ri%d, pk2(%s, %s));", c, c, c, FS(ch.nrs[0]), FS(ch.nrs[1]));
                    S("    float d0l%d, d0h%d; up2(d0%d, d0l%d, d0h%d);", c, c, c, c, c);
                    if (ch.inr[0] && ch.inr[1]) S("    const float dl%d = d0l%d, dh%d = d0h%d; const f32x2 d%d = d0%d;   // always within the cutoff", c, c, c, c, c, c);
                    else {
                        S("    const float dl%d = (r2l%d < K_cutoff2) ? d0l%d : 1.0e18f, dh%d = (r2h%d < K_cutoff2) ? d0h%d : 1.0e18f;", c, c, c, c, c, c);
                        S("    const f32x2 d%d = pk2(dl%d, dh%d);", c, c, c);
                    }
                    S("    const f32x2 aA%d = fma2(mul2(d%d, bc2(-5.770780163555854f)), d%d, bc2(K_lw1));", c, c, c);
                    S("    const f32x2 aB%d = fma2(d%d, fma2(d%d, bc2(-0.36067376022224085f), bc2(2.1640425613334453f)), bc2(K_lw2b));", c, c, c);
                    S("    const f32x2 mn%d = pk2(fminf(dl%d, 0.0f), fminf(dh%d, 0.0f));", c, c, c);
                    S("    const f32x2 c4m%d = mul2(mn%d, bc2(K_c4));", c, c);
                    S("    accR%d = fma2(c4m%d, mn%d, accR%d);", k, c, c, k);
                } else {
                    S("    const float d0%d = fmaf(r2%d, ri%d, %s);", c, c, c, FS(ch.nrs[0]));
                    if (ch.inr[0]) S("    const float d%d = d0%d;", c, c);
                    else S("    const float d%d = (r2%d < K_cutoff2) ? d0%d : 1.0e18f;", c, c, c);
                    S("    const float aA%d = fmaf(d%d * -5.770780163555854f, d%d, K_lw1);", c, c, c);
                    S("    const float aB%d = fmaf(d%d, fmaf(d%d, -0.36067376022224085f, 2.1640425613334453f), K_lw2b);", c, c, c);
                    S("    const float mn%d = fminf(d%d, 0.0f);", c, c);
                    S("    const float c4m%d = mn%d * K_c4;", c, c);
                    S("    sR = fmaf(c4m%d, mn%d, sR);", c, c);
                }
            }
            // stage 4: exponentials
            for (int c = c0; c < c1; ++c) {
                if (chains[c].kind != CH_SCALAR) {
                    S("    float aAl%d, aAh%d, aBl%d, aBh%d; up2(aA%d, aAl%d, aAh%d); up2(aB%d, aBl%d, aBh%d);", c, c, c, c, c, c, c, c, c, c);
                    S("    const f32x2 eA%d = pk2(ex2(aAl%d), ex2(aAh%d)), eB%d = pk2(ex2(aBl%d), ex2(aBh%d));", c, c, c, c, c, c);
                } else
                    S("    const float eA%d = ex2(aA%d), eB%d = ex2(aB%d);", c, c, c, c);
            }
            // stage 5: energies, slopes, forces
            for (int c = c0; c < c1; ++c) {
                const Chain &ch = chains[c];
                const int k = c & 1;
                if (ch.kind != CH_SCALAR) {
                    S("    accA%d = add2(accA%d, eA%d); accB%d = add2(accB%d, eB%d);", k, k, c, k, k, c);
                    S("    f32x2 de%d = fma2(d%d, fma2(bc2(K_q), eB%d, eA%d), fma2(bc2(K_m3q), eB%d, c4m%d));", c, c, c, c, c, c);
                    if (ch.hyd[0] || ch.hyd[1]) {
                        const char *W = (ch.hyd[0] && ch.hyd[1]) ? "WH11" : ch.hyd[0] ? "WH10" : "WH01";
                        S("    { float t0, t1; up2(sub2(bc2(1.5f), d%d), t0, t1); const float h0 = __saturatef(t0), h1 = __saturatef(t1);", c);
                        S("      accH = fma2(%s, pk2(h0, h1), accH); de%d = fma2(%s, pk2((h0 == t0) ? 1.0f : 0.0f, (h1 == t1) ? 1.0f : 0.0f), de%d); }", W, c, W, c);
                    }
                    if (ch.hb[0] || ch.hb[1]) {
                        const char *W = (ch.hb[0] && ch.hb[1]) ? "WB11" : ch.hb[0] ? "WB10" : "WB01";
                        S("    { float t0, t1; up2(mul2(d%d, bc2(-1.4285714285714286f)), t0, t1); const float h0 = __saturatef(t0), h1 = __saturatef(t1);", c);
                        S("      accHB = fma2(%s, pk2(h0, h1), accHB); de%d = fma2(%s, pk2((h0 == t0) ? 1.0f : 0.0f, (h1 == t1) ? 1.0f : 0.0f), de%d); }", W, c, W, c);
                    }
                    if (o.want_grad) {
                        const int t0 = ch.ta[0], t1 = ch.ta[1];
                        S("    { const f32x2 kk = mul2(de%d, ri%d);", c, c);
                        S("      f32x2 tgx = pk2(gx%d, gx%d), tgy = pk2(gy%d, gy%d), tgz = pk2(gz%d, gz%d);", t0, t1, t0, t1, t0, t1);
                        S("      tgx = fma2(kk, dx%d, tgx); tgy = fma2(kk, dy%d, tgy); tgz = fma2(kk, dz%d, tgz);", c, c, c);
                        S("      up2(tgx, gx%d, gx%d); up2(tgy, gy%d, gy%d); up2(tgz, gz%d, gz%d);", t0, t1, t0, t1, t0, t1);
                        if (ch.kind == CH_DIAG) {
                            const int b0 = ch.pa[0], b1 = ch.pa[1];
                            S("      const f32x2 nk = sub2(zero2, kk);");
                            S("      f32x2 bgx = pk2(gx%d, gx%d), bgy = pk2(gy%d, gy%d), bgz = pk2(gz%d, gz%d);", b0, b1, b0, b1, b0, b1);
                            S("      bgx = fma2(nk, dx%d, bgx); bgy = fma2(nk, dy%d, bgy); bgz = fma2(nk, dz%d, bgz);", c, c, c);
                            S("      up2(bgx, gx%d, gx%d); up2(bgy, gy%d, gy%d); up2(bgz, gz%d, gz%d);", b0, b1, b0, b1, b0, b1);
                        } else {
                            S("      float kl, kh, xl, xh, yl, yh, zl, zh; up2(kk, kl, kh); up2(dx%d, xl, xh); up2(dy%d, yl, yh); up2(dz%d, zl, zh);", c, c, c);
                            force_scalar(ch.pa[0], "-", "kl", "xl", "yl", "zl");
                            force_scalar(ch.pa[1], "-", "kh", "xh", "yh", "zh");
                        }
                        S("    }");
                    }
                } else {
                    S("    sA += eA%d; sB += eB%d;", c, c);
                    S("    float de%d = fmaf(d%d, fmaf(K_q, eB%d, eA%d), fmaf(K_m3q, eB%d, c4m%d));", c, c, c, c, c, c);
                    if (ch.hyd[0]) {
                        S("    { const float t0 = 1.5f - d%d, h0 = __saturatef(t0);", c);
                        S("      accH = fma2(WH10, pk2(h0, 0.0f), accH); de%d = fmaf(K_whp, (h0 == t0) ? 1.0f : 0.0f, de%d); }", c, c);
                    }
                    if (ch.hb[0]) {
                        S("    { const float t0 = d%d * -1.4285714285714286f, h0 = __saturatef(t0);", c);
                        S("      accHB = fma2(WB10, pk2(h0, 0.0f), accHB); de%d = fmaf(K_whbp, (h0 == t0) ? 1.0f : 0.0f, de%d); }", c, c);
                    }
                    if (o.want_grad) {
                        char dxn[24], dyn[24], dzn[24];
                        snprintf(dxn, sizeof dxn, "dx%d", c); snprintf(dyn, sizeof dyn, "dy%d", c); snprintf(dzn, sizeof dzn, "dz%d", c);
                        S("    { const float kk = de%d * ri%d;", c, c);
                        force_scalar(ch.ta[0], "", "kk", dxn, dyn, dzn);
                        force_scalar(ch.pa[0], "-", "kk", dxn, dyn, dzn);
                        S("    }");
                    }
                }
            }
        }
        S("    const float sumA = sum2(add2(accA0, accA1)) + sA, sumB = sum2(add2(accB0, accB1)) + sB, sumR = sum2(add2(accR0, accR1)) + sR;");
        S("    const float e_intra = fmaf(K_eA, sumA, fmaf(K_eB, sumB, K_sigma * fmaf(0.5f, sumR, fmaf(-0.7f, sum2(accHB), -sum2(accH)))));");
    }

    void chain_rule()
    {
        const int T = d.T;
        const int CR = 1000000;                             // group tag of the loads of this phase
        last_load.assign(d.D, -100);
        S("    // ---- phases 3 + 4: A5 (sigma-scaled until the stores) ----");
        int s = 0;
        for (int f = 0; f <= T; ++f) {
            if (f > 0) {
                const int bs = d.tors[f - 1].b_slot;
                need_duo(duo_of[bs], CR);
                S("    const float o%d_x = %s, o%d_y = %s, o%d_z = %s;", f, sx(bs).c_str(), f, sy(bs).c_str(), f, sz(bs).c_str());
            } else
                S("    const float o0_x = 0.0f, o0_y = 0.0f, o0_z = 0.0f;");
            S("    float F%d_x = 0.0f, F%d_y = 0.0f, F%d_z = 0.0f, M%d_x = 0.0f, M%d_y = 0.0f, M%d_z = 0.0f;", f, f, f, f, f, f);
            for (; s < d.frag_end[f]; ++s) {
                need_duo(duo_of[s], CR);
                S("    { const float lx = %s - o%d_x, ly = %s - o%d_y, lz = %s - o%d_z;", sx(s).c_str(), f, sy(s).c_str(), f, sz(s).c_str(), f);
                S("      F%d_x += gx%d; F%d_y += gy%d; F%d_z += gz%d;", f, s, f, s, f, s);
                S("      M%d_x = fmaf(ly, gz%d, fmaf(-lz, gy%d, M%d_x)); M%d_y = fmaf(lz, gx%d, fmaf(-lx, gz%d, M%d_y)); M%d_z = fmaf(lx, gy%d, fmaf(-ly, gx%d, M%d_z)); }",
                  f, s, s, f, f, s, s, f, f, s, s, f);
            }
        }
        for (int f = T; f >= 1; --f) {
            const JitTors &t = d.tors[f - 1];
            need_duo(duo_of[t.a_slot], CR);
            need_duo(duo_of[t.b_slot], CR);
            S("    {");
            S("        const float xbx = %s, xby = %s, xbz = %s;", sx(t.b_slot).c_str(), sy(t.b_slot).c_str(), sz(t.b_slot).c_str());
            S("        const float w = %s * K_sigma;", FS(t.inv_len));
            S("        const float ux = (xbx - %s) * w, uy = (xby - %s) * w, uz = (xbz - %s) * w;", sx(t.a_slot).c_str(), sy(t.a_slot).c_str(), sz(t.a_slot).c_str());
            S("        OUT(grad + %d, fmaf(ux, M%d_x, fmaf(uy, M%d_y, uz * M%d_z)));", 6 + f - 1, f, f, f);
            const int p = t.parent;
            if (p > 0) {
                S("        const float lx = xbx - o%d_x, ly = xby - o%d_y, lz = xbz - o%d_z;", p, p, p);
                S("        M%d_x += M%d_x + fmaf(ly, F%d_z, -lz * F%d_y);", p, f, f, f);
                S("        M%d_y += M%d_y + fmaf(lz, F%d_x, -lx * F%d_z);", p, f, f, f);
                S("        M%d_z += M%d_z + fmaf(lx, F%d_y, -ly * F%d_x);", p, f, f, f);
            } else {
                S("        M0_x += M%d_x + fmaf(xby, F%d_z, -xbz * F%d_y);", f, f, f);
                S("        M0_y += M%d_y + fmaf(xbz, F%d_x, -xbx * F%d_z);", f, f, f);
                S("        M0_z += M%d_z + fmaf(xbx, F%d_y, -xby * F%d_x);", f, f, f);
            }
            S("        F%d_x += F%d_x; F%d_y += F%d_y; F%d_z += F%d_z;", p, f, p, f, p, f);
            S("    }");
        }
        S("    OUT(grad + 0, K_sigma * F0_x); OUT(grad + 1, K_sigma * F0_y); OUT(grad + 2, K_sigma * F0_z);");
        S("    OUT(grad + 3, K_sigma * M0_x); OUT(grad + 4, K_sigma * M0_y); OUT(grad + 5, K_sigma * M0_z);");
    }

    std::string run()
    {
        choose_duos();
        S("// generated by libdock_b200 (jit_score.cu): N = %d, T = %d, P = %zu, grad = %d", d.N, d.T, d.pairs.size(), (int)o.want_grad);
        S("struct JitArgs { %s };", DOCK_JIT_STR(DOCK_JIT_ARGS_BODY));
        S("#define JIT_QUAD %d", o.quad ? 1 : 0);
        if (o.stream) {                                   // poses and outputs pass through L2 once: streaming hints keep the maps in
            S("#define POSE(k) __ldcs(pose + (k))");
            S("#define OUT(ptr, v) __stcs(ptr, v)");
        } else {
            S("#define POSE(k) pose[k]");
            S("#define OUT(ptr, v) (*(ptr) = (v))");
        }
        S.s += k_prelude;
        S.s += tables();
        S("extern \"C\" __global__ void __launch_bounds__(%d, %d) dock_score_jit(const JitArgs a)", 32 * o.warps, o.min_blocks);
        S("{");
        S("    extern __shared__ float4 smem4[];");
        S("    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;");
        // per warp: [xyq: D x 32 float4][zq: D x 32 float2][region 2: frames [T][6] float2 x 32 in phase 1, then
        //            gq4: D x 32 float4, gq2: D x 32 float2 (grid forces)]
        const int per_warp4 = jit_warp_float4(d.N, d.T, o.want_grad != 0);
        S("    float4 *const xyq = smem4 + warp * %d + lane;", per_warp4);
        S("    float2 *const zq = reinterpret_cast<float2 *>(smem4 + warp * %d + %d) + lane;", per_warp4, d.D * 32);
        S("    float4 *const reg2 = smem4 + warp * %d + %d;", per_warp4, d.D * 48);
        if (o.want_grad) {
            S("    float4 *const gq4 = reg2 + lane;");
            S("    float2 *const gq2 = reinterpret_cast<float2 *>(reg2 + %d) + lane;", d.D * 32);
        }
        S("    long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;");
        S("    if (p > a.n_poses - 1) p = a.n_poses - 1;   // idle lanes of the last warp redo the last pose (same bits, same stores)");
        S("    const float *__restrict__ pose = a.poses + p * %d;", 7 + d.T);
        if (o.want_grad) S("    float *__restrict__ grad = a.grad + p * %d;", 6 + d.T);
        if (o.quad) {
            S("    const float4 *__restrict__ maps = reinterpret_cast<const float4 *>(a.packed);");
            S("#define LDG_CELL(ptr, lo, hi) ldg_quad(ptr, lo, hi)");
        } else
            S("    const Cell8 *__restrict__ maps = reinterpret_cast<const Cell8 *>(a.packed);");
        if (o.quad) {
        } else if (o.l2_hint) {
            S("    unsigned long long l2_keep; asm volatile(\"createpolicy.fractional.L2::evict_last.b64 %%0, 1.0;\" : \"=l\"(l2_keep));");
            S("#define LDG_CELL(ptr, lo, hi) ldg_cell_hint(ptr, lo, hi, l2_keep)");
        } else
            S("#define LDG_CELL(ptr, lo, hi) ldg_cell(ptr, lo, hi)");
        S("    constexpr float K_cutoff2 = %s, K_lw2b = %s, K_q = %s, K_m3q = %s, K_c4 = %s, K_sigma = %s, K_eA = %s, K_eB = %s;",
          k_cutoff2.c_str(), k_lw2b.c_str(), k_q.c_str(), k_m3q.c_str(), k_c4.c_str(), k_sigma.c_str(), k_eA.c_str(), k_eB.c_str());
        S("    const float K_lw1 = %s, K_whp = %s, K_whbp = %s;", k_lw1.c_str(), k_whp.c_str(), k_whbp.c_str());
        S("    const float tx = (POSE(0) - a.rx) - a.rdx, ty = (POSE(1) - a.ry) - a.rdy, tz = (POSE(2) - a.rz) - a.rdz;");
        kinematics();
        grid_loop();
        pair_phase();
        if (o.want_grad) chain_rule();
        S("    OUT(a.energy + p, e_grid + e_wall + e_intra);");
        S("    if (a.terms) { OUT(a.terms + 3 * p, e_grid); OUT(a.terms + 3 * p + 1, e_wall); OUT(a.terms + 3 * p + 2, e_intra); }");
        S("}");
        return S.s;
    }
};

// ---- NVRTC through dlopen ----------------------------------------------------------------------------
typedef struct _nvrtcProgram *nvrtcProgram;
struct Nvrtc {
    void *h = nullptr;
    int (*CreateProgram)(nvrtcProgram *, const char *, const char *, int, const char *const *, const char *const *) = nullptr;
    int (*CompileProgram)(nvrtcProgram, int, const char *const *) = nullptr;
    int (*GetCUBINSize)(nvrtcProgram, size_t *) = nullptr;
    int (*GetCUBIN)(nvrtcProgram, char *) = nullptr;
    int (*GetProgramLogSize)(nvrtcProgram, size_t *) = nullptr;
    int (*GetProgramLog)(nvrtcProgram, char *) = nullptr;
    int (*DestroyProgram)(nvrtcProgram *) = nullptr;
    bool ok = false;
};

Nvrtc &nvrtc()
{
    static Nvrtc n;
    static std::once_flag once;
    std::call_once(once, [] {
        // the 256-bit map load (ld.global.nc.v4.b64) needs the PTX ISA of CUDA 12.9: a process may already hold an older
        // libnvrtc.so.12 (PyTorch ships one), so the toolkit's own copy is tried first and the version is checked
        const char *names[] = {"/usr/local/cuda/lib64/libnvrtc.so.12", "/usr/local/cuda/lib64/libnvrtc.so", "libnvrtc.so.12", "libnvrtc.so"};
        for (const char *nm : names) {
            void *h = dlopen(nm, RTLD_NOW | RTLD_LOCAL);
            if (!h) continue;
            int (*ver)(int *, int *) = nullptr;
            *(void **)(&ver) = dlsym(h, "nvrtcVersion");
            int major = 0, minor = 0;
            if (ver && ver(&major, &minor) == 0 && (major > 12 || (major == 12 && minor >= 9))) { n.h = h; break; }
            dlclose(h);
        }
        if (!n.h) return;
#define DOCK_NVRTC_SYM(field, sym) *(void **)(&n.field) = dlsym(n.h, sym)
        DOCK_NVRTC_SYM(CreateProgram, "nvrtcCreateProgram");
        DOCK_NVRTC_SYM(CompileProgram, "nvrtcCompileProgram");
        DOCK_NVRTC_SYM(GetCUBINSize, "nvrtcGetCUBINSize");
        DOCK_NVRTC_SYM(GetCUBIN, "nvrtcGetCUBIN");
        DOCK_NVRTC_SYM(GetProgramLogSize, "nvrtcGetProgramLogSize");
        DOCK_NVRTC_SYM(GetProgramLog, "nvrtcGetProgramLog");
        DOCK_NVRTC_SYM(DestroyProgram, "nvrtcDestroyProgram");
#undef DOCK_NVRTC_SYM
        n.ok = n.CreateProgram && n.CompileProgram && n.GetCUBINSize && n.GetCUBIN && n.GetProgramLogSize && n.GetProgramLog && n.DestroyProgram;
    });
    return n;
}

std::string g_jit_log;                                   // log of the last failed compilation (dock_score_jit_log)
std::mutex g_jit_mu;

int compile_cubin(const std::string &src, const JitOpts &o, std::vector<char> &cubin)
{
    Nvrtc &n = nvrtc();
    if (!n.ok) { g_jit_log = "no libnvrtc.so.12 of CUDA >= 12.9 found"; return DOCK_ECUDA; }
    nvrtcProgram prog = nullptr;
    if (n.CreateProgram(&prog, src.c_str(), "dock_score_jit.cu", 0, nullptr, nullptr) != 0) return DOCK_ECUDA;
    std::vector<const char *> opts = {"--gpu-architecture=sm_100a", "--std=c++17", "-lineinfo", "--fmad=true"};
    char mr[64];
    if (o.maxrreg > 0) { snprintf(mr, sizeof mr, "--maxrregcount=%d", o.maxrreg); opts.push_back(mr); }
    const int rc = n.CompileProgram(prog, (int)opts.size(), opts.data());
    if (rc != 0) {
        size_t ls = 0;
        n.GetProgramLogSize(prog, &ls);
        g_jit_log.assign(ls, '\0');
        if (ls) n.GetProgramLog(prog, &g_jit_log[0]);
        n.DestroyProgram(&prog);
        return DOCK_ECUDA;
    }
    size_t cs = 0;
    n.GetCUBINSize(prog, &cs);
    cubin.resize(cs);
    n.GetCUBIN(prog, cubin.data());
    n.DestroyProgram(&prog);
    return DOCK_OK;
}

struct JitKernel {
    cudaLibrary_t lib = nullptr;
    cudaKernel_t kern = nullptr;
    int warps = 0;
    size_t smem = 0;
    int status = DOCK_OK;                 // a failed compilation is remembered: no retry storm
    uint64_t last_use = 0;                // g_cache_tick at the last launch: the least recently used entry is evicted
};
// (device, digest of everything the generated text depends on) -> kernel.  Bounded per device (a screening run sees
// thousands of ligands): at g_cache_limit entries the least recently used one of that device is unloaded first.
std::map<std::pair<int, std::pair<uint64_t, uint64_t>>, JitKernel> g_cache;
uint64_t g_cache_tick = 0;
int g_cache_limit = 64;

// Called under g_jit_mu before an entry for `dev` is added.  The victim's kernel may still be running on some stream of the
// device, so the device is synchronised before cudaLibraryUnload; this happens only next to a compilation (0.4-6 s).
void jit_cache_make_room(int dev)
{
    for (;;) {
        int n = 0;
        auto victim = g_cache.end();
        for (auto it = g_cache.begin(); it != g_cache.end(); ++it) {
            if (it->first.first != dev) continue;
            ++n;
            if (victim == g_cache.end() || it->second.last_use < victim->second.last_use) victim = it;
        }
        if (n < g_cache_limit || victim == g_cache.end()) return;
        if (victim->second.lib) {
            cudaDeviceSynchronize();
            cudaLibraryUnload(victim->second.lib);
        }
        g_cache.erase(victim);
    }
}

struct Digest {                                            // two independent 64-bit FNV-1a style streams
    uint64_t a = 1469598103934665603ull, b = 0x9e3779b97f4a7c15ull;
    void add(const void *p, size_t n)
    {
        const unsigned char *c = (const unsigned char *)p;
        for (size_t i = 0; i < n; ++i) {
            a = (a ^ c[i]) * 1099511628211ull;
            b = (b + c[i] + 0x7f4a7c15ull) * 0xd6e8feb86659fd93ull; b ^= b >> 29;
        }
    }
};

std::pair<uint64_t, uint64_t> jit_key(const dock_params *p, const dock_grid *g, const dock_ligand *L, const JitOpts &o)
{
    Digest d;
    d.add(&o, sizeof o);
    d.add(p->radius, sizeof p->radius); d.add(p->hydrophobic, sizeof p->hydrophobic);
    d.add(p->donor, sizeof p->donor); d.add(p->acceptor, sizeof p->acceptor);
    d.add(p->w, sizeof p->w); d.add(&p->cutoff, sizeof p->cutoff); d.add(&p->n_types, sizeof p->n_types);
    d.add(g->type_to_map, sizeof g->type_to_map);
    d.add(&L->N, sizeof(int)); d.add(&L->T, sizeof(int)); d.add(&L->P, sizeof(int));
    d.add(L->ref_xyz, sizeof(float) * 3 * L->N); d.add(L->type, sizeof(int) * L->N); d.add(L->atom_fragment, sizeof(int) * L->N);
    if (L->T > 0) { d.add(L->tors_parent, sizeof(int) * L->T); d.add(L->tors_a, sizeof(int) * L->T); d.add(L->tors_b, sizeof(int) * L->T); }
    if (L->P > 0) d.add(L->pairs, sizeof(int) * 2 * L->P);
    return {d.a, d.b};
}

}  // namespace

JitOpts jit_default_opts()
{
    JitOpts o;
    o.want_grad = true;
    o.group = 4;
    o.warps = 4;
    o.min_blocks = 2;
    o.maxrreg = 0;
    o.sync_every = 0;
    o.reuse = 1;
    o.grid_unroll = 1;
    o.grid_sets = 2;
    o.stream = 1;
    o.quad = 1;
    o.l2_hint = 0;           // measured: 0.925 ms with evict_last on the gathers, 0.838 ms without; the L2 hit rate stays 46 %
    o.prefetch = 0;          // measured: 0.853-0.873 ms with it, 0.841 ms without (configs[1])
    o.atom_unroll = 2;
    if (const char *e = getenv("DOCK_JIT_TUNE")) {        // tuning aid, e.g. "group=6,warps=8,minb=1,gu=2,reuse=2"
        int v;
        const char *q;
        if ((q = strstr(e, "group=")) && sscanf(q + 6, "%d", &v) == 1 && v >= 1 && v <= 16) o.group = v;
        if ((q = strstr(e, "warps=")) && sscanf(q + 6, "%d", &v) == 1 && v >= 1 && v <= 32) o.warps = v;
        if ((q = strstr(e, "minb=")) && sscanf(q + 5, "%d", &v) == 1 && v >= 1 && v <= 16) o.min_blocks = v;
        if ((q = strstr(e, "maxrreg=")) && sscanf(q + 8, "%d", &v) == 1 && v >= 0 && v <= 255) o.maxrreg = v;
        if ((q = strstr(e, "sync=")) && sscanf(q + 5, "%d", &v) == 1 && v >= 0 && v <= 1024) o.sync_every = v;
        if ((q = strstr(e, "st=")) && sscanf(q + 3, "%d", &v) == 1 && v >= 0 && v <= 1) o.stream = v;
        if ((q = strstr(e, "quad=")) && sscanf(q + 5, "%d", &v) == 1 && v >= 0 && v <= 1) o.quad = v;
        if ((q = strstr(e, "l2=")) && sscanf(q + 3, "%d", &v) == 1 && v >= 0 && v <= 1) o.l2_hint = v;
        if ((q = strstr(e, "pf=")) && sscanf(q + 3, "%d", &v) == 1 && v >= 0 && v <= 1) o.prefetch = v;
        if ((q = strstr(e, "gs=")) && sscanf(q + 3, "%d", &v) == 1 && v >= 2 && v <= 6) o.grid_sets = v;
        if ((q = strstr(e, "au=")) && sscanf(q + 3, "%d", &v) == 1 && v >= 1 && v <= 8) o.atom_unroll = v;
        if ((q = strstr(e, "gu=")) && sscanf(q + 3, "%d", &v) == 1 && v >= 1 && v <= 8) o.grid_unroll = v;
        if ((q = strstr(e, "reuse=")) && sscanf(q + 6, "%d", &v) == 1 && v >= 0 && v <= 1000) o.reuse = v;
    }
    return o;
}

int jit_score_source(const dock_params *p, const dock_grid *g, const dock_ligand *L, const JitOpts &o, std::string &out)
{
    if (!p || !g || !L) return DOCK_EINVAL;
    if (L->N > DOCK_JIT_MAX_ATOMS || g->n_channels == 4) return DOCK_EINVAL;
    JitDesc d;
    if (build_desc(p, g, L, d) != DOCK_OK) return DOCK_EINVAL;
    DevParams P;
    if (dock_make_dev_params(p, &P) != DOCK_OK) return DOCK_EINVAL;
    Gen gen(d, o);
    gen.set_params(p, P);
    out = gen.run();
    return DOCK_OK;
}

int jit_score_launch(const dock_params *p, const dock_grid *g, const dock_ligand *L, const DevParams &P, const DevGrid &G,
                     long long n_poses, const float *poses_dev, float *energy_dev, float *grad_dev, float *terms_dev,
                     cudaStream_t stream)
{
    if (!p || !g || !L || L->N < 1 || L->N > DOCK_JIT_MAX_ATOMS || L->T < 0 || L->P < 0 || g->n_channels == 4) return DOCK_EINVAL;
    if (!L->ref_xyz || !L->type || !L->atom_fragment || (L->T > 0 && (!L->tors_parent || !L->tors_a || !L->tors_b)) || (L->P > 0 && !L->pairs))
        return DOCK_EINVAL;
    JitOpts o = jit_default_opts();
    o.want_grad = grad_dev != nullptr;
    int dev = 0;
    DOCK_CUDA_CHECK(cudaGetDevice(&dev));
    JitKernel k;
    {
        std::lock_guard<std::mutex> lock(g_jit_mu);
        auto key = std::make_pair(dev, jit_key(p, g, L, o));
        auto it = g_cache.find(key);
        if (it == g_cache.end()) {
            JitKernel nk;
            std::vector<char> cubin;
            std::string src;
            nk.status = jit_score_source(p, g, L, o, src);      // validates the ligand
            if (nk.status == DOCK_OK) nk.status = compile_cubin(src, o, cubin);
            if (nk.status == DOCK_OK) {
                cudaError_t e = cudaLibraryLoadData(&nk.lib, cubin.data(), nullptr, nullptr, 0, nullptr, nullptr, 0);
                if (e == cudaSuccess) e = cudaLibraryGetKernel(&nk.kern, nk.lib, "dock_score_jit");
                nk.warps = o.warps;
                nk.smem = (size_t)o.warps * jit_warp_float4(L->N, L->T, o.want_grad != 0) * 16;
                if (e == cudaSuccess && nk.smem > 48 * 1024)
                    e = cudaFuncSetAttribute((const void *)nk.kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)nk.smem);
                if (e != cudaSuccess) { g_dock_last_cuda_error.store((int)e); nk.status = DOCK_ECUDA; }
            }
            jit_cache_make_room(dev);
            it = g_cache.emplace(key, nk).first;
        }
        it->second.last_use = ++g_cache_tick;
        k = it->second;
    }
    if (k.status != DOCK_OK) return k.status;
    if (o.quad && !g->quad_dev) return DOCK_EINVAL;        // descriptor without the 4-corner image (dock.h: dock_grid.quad_dev)
    JitArgs a;
    a.nx = G.nx; a.ny = G.ny; a.nz = G.nz; a.icx = G.icx; a.icy = G.icy; a.icz = G.icz;
    a.rx = G.rx; a.ry = G.ry; a.rz = G.rz; a.rdx = G.rdx; a.rdy = G.rdy; a.rdz = G.rdz;
    a.lo_x = G.lo_x; a.lo_y = G.lo_y; a.lo_z = G.lo_z; a.hi_x = G.hi_x; a.hi_y = G.hi_y; a.hi_z = G.hi_z;
    a.inv_h = G.inv_h; a.inv_h_lo = G.inv_h_lo; a.kw_g = G.kw_g; a.kw_e = G.kw_e;
    a.map_stride = (long long)G.chan_stride * G.channels;
    a.packed = o.quad ? (const void *)g->quad_dev : (const void *)G.packed;
    a.n_poses = n_poses; a.poses = poses_dev; a.energy = energy_dev; a.grad = grad_dev; a.terms = terms_dev;
    const long long per_cta = 32LL * k.warps;
    const long long blocks = (n_poses + per_cta - 1) / per_cta;
    if (blocks > 0x7fffffffLL) return DOCK_EINVAL;
    void *args[] = {&a};
    DOCK_CUDA_CHECK(cudaLaunchKernel((const void *)k.kern, dim3((unsigned)blocks), dim3((unsigned)per_cta), args, k.smem, stream));
    g_dock_launches.fetch_add(1);
    return DOCK_OK;
}

bool jit_available() { return nvrtc().ok; }

extern "C" int dock_score_jit_source(const dock_params *params, const dock_grid *grid, const dock_ligand *ligand,
                                     int32_t want_grad, char *buf, size_t cap, size_t *needed)
{
    JitOpts o = jit_default_opts();
    o.want_grad = want_grad != 0;
    std::string src;
    const int rc = jit_score_source(params, grid, ligand, o, src);
    if (rc != DOCK_OK) return rc;
    if (needed) *needed = src.size() + 1;
    if (!buf || cap < src.size() + 1) return DOCK_EWORKSPACE;
    std::memcpy(buf, src.c_str(), src.size() + 1);
    return DOCK_OK;
}

extern "C" int dock_score_jit_compile(const dock_params *params, const dock_grid *grid, const dock_ligand *ligand,
                                      int32_t want_grad, size_t *cubin_bytes)
{
    JitOpts o = jit_default_opts();
    o.want_grad = want_grad != 0;
    std::string src;
    const int rc = jit_score_source(params, grid, ligand, o, src);
    if (rc != DOCK_OK) return rc;
    std::lock_guard<std::mutex> lock(g_jit_mu);
    std::vector<char> cubin;
    const int rc2 = compile_cubin(src, o, cubin);
    if (cubin_bytes) *cubin_bytes = cubin.size();
    return rc2;
}

extern "C" int dock_score_jit_cache(int32_t new_limit, int32_t *old_limit, int32_t *entries)
{
    std::lock_guard<std::mutex> lock(g_jit_mu);
    if (old_limit) *old_limit = g_cache_limit;
    if (entries) *entries = (int32_t)g_cache.size();
    if (new_limit < 0) return DOCK_OK;
    if (new_limit < 1 || new_limit > 65536) return DOCK_EINVAL;
    g_cache_limit = new_limit;
    return DOCK_OK;
}

extern "C" const char *dock_score_jit_log(void)
{
    std::lock_guard<std::mutex> lock(g_jit_mu);
    static std::string copy;
    copy = g_jit_log;
    return copy.c_str();
}
