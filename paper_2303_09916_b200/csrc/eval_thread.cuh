// eval_thread.cuh -- fused pose -> coordinates -> energy + gradient, ONE THREAD PER POSE
// (eq. 2-3 at 198-219).  The throughput evaluator behind
// dock_score_batch.
//
// Why one thread per pose: all poses of a batch share the ligand, so the pair list, the torsion tree
// and every per-type constant are warp-uniform.  They live in the kernel-parameter constant bank
// (TppLigand) and are read with uniform 128-bit constant loads; control flow is uniform, there are
// no shuffles, no barriers and no idle lanes.  Per-thread state that needs dynamic indexing
// (coordinates, per-atom forces, fragment frames, per-fragment force/torque) sits in shared memory
// as [row][lane] columns: conflict-free, thread-private, so no synchronisation at all.
//
// Shared memory (6N floats per pose) and registers bound the occupancy (8 warps per SM for a 30-atom
// ligand), so the kernel is written for instruction-level parallelism instead: the pair phase is
// branch-free straight-line code over 8 independent pairs (2 partner atoms x a 4-atom register tile),
// written stage by stage on packed fp32x2 register pairs (two tile atoms per FFMA2 issue slot), and
// the 32-byte map gathers of a tile's atoms are issued at the top of the tile's pair group and
// consumed at its end, so their L2 latency hides under the pair arithmetic
// (profiles/r1a.md -> r1f.md -> r1j.md).
//
//   phase 1  A2: one rigid frame (rotation + offset) per fragment, parents first, composed from the
//            parent's frame and one Rodrigues rotation; atoms of a fragment are 9 FMAs each.
//            Coordinates are stored RELATIVE TO THE PIVOT (smaller numbers -> smaller fp32 error in
//            pair distances and lever arms); the translation is added for the grid lookup only.
//   phase 2  A3 + A4, one group per tile of 4 atoms: issue the tile's map gathers; intra-ligand
//            pair records of the tile (schedule format: common.cuh; weights folded into the
//            exponent arguments, unlisted pairs masked through their data, forces carried
//            sigma-scaled, see DevParams); trilinear energy + gradient + wall of the tile's atoms.
//   phase 3  A5: per-fragment force / torque sums about the fragment's origin
//   phase 4  A5: up-sweep over the torsion tree (children before parents): dE/dtheta_k = u_k . M_k,
//            then the fragment's force / torque are folded into its parent's (the root's stay in registers)
#pragma once

#include "common.cuh"
#include "mathx.cuh"

struct EvalTerms {
    float e_grid, e_wall, e_intra;
};

// floats of shared memory one THREAD of the evaluator needs:
//   [xy: 2N][z: N][R: max(3N, 12 T)  per-atom forces, aliased by the fragment frames in phase 1][fm: 6 T unless aliased]
// fm (force / torque sums of fragments 1..T) aliases the force slots of atoms 2(f-1), 2(f-1)+1 when the host
// found that those atoms are consumed before fragment f's sums are written (TppLigand::fm_alias).
__host__ __device__ inline int tpp_thread_floats(int N, int T, bool want_grad, bool fm_alias)
{
    const int frames = 12 * T;
    if (!want_grad) return 3 * N + frames;
    return 3 * N + (3 * N > frames ? 3 * N : frames) + (fm_alias ? 0 : 6 * T);
}
__host__ __device__ inline int tpp_warp_floats(int N, int T, bool want_grad, bool fm_alias)
{
    return 32 * tpp_thread_floats(N, T, want_grad, fm_alias);
}

template <bool SCHED_PARAM>
__device__ __forceinline__ uint4 tpp_quad(const TppLigand &L, int pos)
{
    return SCHED_PARAM ? L.sched[pos] : __ldg(L.sched_global + pos);
}

// Accumulators of the pair phase (DevParams): E_intra = eA a + eB b + sigma/2 rep - sigma hyd - 0.7 sigma hb.
// Packed pairs: the two halves belong to tile atoms (0,1) / (2,3) and are added at the very end.
struct PairAcc {
    f32x2 a, b, rep, hyd, hb;
};

// The register tile of the pair phase: TPP_TILE = 4 atoms as two packed halves h = 0: atoms (0,1), h = 1: atoms
// (2,3), with their force accumulators.
struct PairTile {
    f32x2 x[2], y[2], z[2], fx[2], fy[2], fz[2];
};

__device__ __forceinline__ void quad_halves(const uint4 q, f32x2 v[2])
{
    v[0] = pk2(__uint_as_float(q.x), __uint_as_float(q.y));
    v[1] = pk2(__uint_as_float(q.z), __uint_as_float(q.w));
}

// A partner atom's coordinates and force accumulator, read one record ahead (record_class).
struct PartnerRegs { float x, y, z, gx, gy, gz; };

template <bool WANT_GRAD>
__device__ __forceinline__ void load_partner(unsigned off, const char *xy, const char *zz, char *gxy, char *gz, PartnerRegs &p)
{
    // volatile: keeps the loads where they are written (ahead of the arithmetic of the previous record)
    const unsigned axy = (unsigned)__cvta_generic_to_shared(xy + 2 * off), az = (unsigned)__cvta_generic_to_shared(zz + off);
    asm volatile("ld.volatile.shared.v2.f32 {%0,%1}, [%2];" : "=f"(p.x), "=f"(p.y) : "r"(axy));
    asm volatile("ld.volatile.shared.f32 %0, [%1];" : "=f"(p.z) : "r"(az));
    p.gx = p.gy = p.gz = 0.0f;
    if (WANT_GRAD) {
        const unsigned bxy = (unsigned)__cvta_generic_to_shared(gxy + 2 * off), bz = (unsigned)__cvta_generic_to_shared(gz + off);
        asm volatile("ld.volatile.shared.v2.f32 {%0,%1}, [%2];" : "=f"(p.gx), "=f"(p.gy) : "r"(bxy));
        asm volatile("ld.volatile.shared.f32 %0, [%1];" : "=f"(p.gz) : "r"(bz));
    }
}

// One record block: NP partner atoms (1 or 2) against the 4 tile atoms = 4 NP pairs, written STAGE BY STAGE over
// all pairs (distances; reciprocal square roots; surface distances and exponent arguments; exponentials; slopes
// and forces) so that the multi-cycle MUFU results of one pair are produced while the others issue -- with two
// warps per scheduler the latency has to be hidden inside the warp (profiles/r1d.md).
//   Pair (i, j): d = r - rsum; accumulates the energy terms and the sigma-scaled force k (x_i - x_j) on i, -that
//   on j.  rsum = TPP_MASKED_RSUM makes every term exactly 0.  CLS 1 adds the hydrophobic ramp, CLS 2 the
//   hydrophobic and H-bond ramps, with the per-pair weights wh', whb' (0 where the type pair has none).
// Partner columns sit at byte offset `off` (z column; the (x,y) column is at 2*off).
template <int NP, int CLS, bool WANT_GRAD, bool SCHED_PARAM, bool PRE = false>
__device__ __forceinline__ void record_block(const DevParams &P, const TppLigand &L, int &pos, PairTile &t, PairAcc *acc,
                                             const char *xy, const char *zz, char *gxy, char *gz,
                                             const PartnerRegs *pre = nullptr)
{
    constexpr int S = 1 + CLS;                 // payload quads of one record
    constexpr int NC = NP * 2;                 // packed chains of the block; chain c = partner c / 2, tile half c % 2
    const uint4 h = tpp_quad<SCHED_PARAM>(L, pos);
    const unsigned off[2] = {h.x, h.y};
    f32x2 nrs[NC], wh[NC], wb[NC];
#pragma unroll
    for (int a = 0; a < NP; ++a) {
        quad_halves(tpp_quad<SCHED_PARAM>(L, pos + 1 + a * S), nrs + 2 * a);
        if (CLS >= 1) quad_halves(tpp_quad<SCHED_PARAM>(L, pos + 2 + a * S), wh + 2 * a);
        if (CLS >= 2) quad_halves(tpp_quad<SCHED_PARAM>(L, pos + 3 + a * S), wb + 2 * a);
    }
    pos += 1 + NP * S;
    float jx[NP], jy[NP], jz[NP];
#pragma unroll
    for (int a = 0; a < NP; ++a) {
        if (PRE) { jx[a] = pre[a].x; jy[a] = pre[a].y; jz[a] = pre[a].z; }
        else {
            const float2 c = *reinterpret_cast<const float2 *>(xy + 2 * off[a]);
            jx[a] = c.x; jy[a] = c.y; jz[a] = *reinterpret_cast<const float *>(zz + off[a]);
        }
    }
    f32x2 dx[NC], dy[NC], dz[NC], r2[NC], rinv[NC], d[NC], argA[NC], argB[NC], c4m[NC], eA[NC], eB[NC];
#pragma unroll
    for (int c = 0; c < NC; ++c) {
        const int a = c / 2, hf = c % 2;
        dx[c] = sub2(t.x[hf], bc2(jx[a])); dy[c] = sub2(t.y[hf], bc2(jy[a])); dz[c] = sub2(t.z[hf], bc2(jz[a]));
        r2[c] = fma2(dz[c], dz[c], fma2(dy[c], dy[c], fma2(dx[c], dx[c], bc2(1e-12f))));
    }
#pragma unroll
    for (int c = 0; c < NC; ++c) {
        float r0, r1;
        up2(r2[c], r0, r1);
        rinv[c] = pk2(fast_rsqrt(r0), fast_rsqrt(r1));
    }
#pragma unroll
    for (int c = 0; c < NC; ++c) {
        const int a = c / 2;
        // out of range (r >= cutoff, decided on r^2 in fp32) -> the same "infinitely far" surface distance as a
        // masked pair: every term and derivative below is then exactly 0, with no branch in the instruction stream
        const f32x2 d0 = fma2(r2[c], rinv[c], nrs[c]);
        float r0, r1, d0l, d0h;
        up2(r2[c], r0, r1);
        up2(d0, d0l, d0h);
        const float dl = (r0 < P.cutoff2) ? d0l : 1.0e18f, dh = (r1 < P.cutoff2) ? d0h : 1.0e18f;
        d[c] = pk2(dl, dh);
        argA[c] = fma2(mul2(d[c], bc2(-5.770780163555854f)), d[c], bc2(P.lw1));  // log2 of 8|w1| exp(-(d/0.5)^2)
        // -log2(e)/4 (d-3)^2 + lw2 expanded in d
        argB[c] = fma2(d[c], fma2(d[c], bc2(-0.36067376022224085f), bc2(2.1640425613334453f)), bc2(P.lw2 - 3.2460638420001677f));
        const f32x2 m = pk2(fminf(dl, 0.0f), fminf(dh, 0.0f));
        c4m[c] = mul2(m, bc2(P.c4));
        acc[a].rep = fma2(c4m[c], m, acc[a].rep);
    }
#pragma unroll
    for (int c = 0; c < NC; ++c) {
        float a0, a1, b0, b1;
        up2(argA[c], a0, a1);
        up2(argB[c], b0, b1);
        eA[c] = pk2(fast_ex2(a0), fast_ex2(a1));
        eB[c] = pk2(fast_ex2(b0), fast_ex2(b1));
    }
    f32x2 gx[NP], gy[NP], gzz[NP];                 // force on the partner, sign flipped (subtracted at the end)
#pragma unroll
    for (int a = 0; a < NP; ++a) gx[a] = gy[a] = gzz[a] = bc2(0.0f);
#pragma unroll
    for (int c = 0; c < NC; ++c) {
        const int a = c / 2, hf = c % 2;
        acc[a].a = add2(acc[a].a, eA[c]);
        acc[a].b = add2(acc[a].b, eB[c]);
        f32x2 de = fma2(d[c], fma2(bc2(P.q), eB[c], eA[c]), fma2(bc2(P.m3q), eB[c], c4m[c]));   // sigma dE/dd
        if (CLS >= 1) {
            float t0, t1;
            up2(sub2(bc2(1.5f), d[c]), t0, t1);                                   // hydrophobic: 1 | 1.5 - d | 0
            const float h0 = __saturatef(t0), h1 = __saturatef(t1);
            acc[a].hyd = fma2(wh[c], pk2(h0, h1), acc[a].hyd);
            de = fma2(wh[c], pk2((h0 == t0) ? 1.0f : 0.0f, (h1 == t1) ? 1.0f : 0.0f), de);   // on the ramp iff the clamp did nothing
        }
        if (CLS >= 2) {
            float t0, t1;
            up2(mul2(d[c], bc2(-1.4285714285714286f)), t0, t1);                   // H-bond: 1 | -d/0.7 | 0
            const float h0 = __saturatef(t0), h1 = __saturatef(t1);
            acc[a].hb = fma2(wb[c], pk2(h0, h1), acc[a].hb);
            de = fma2(wb[c], pk2((h0 == t0) ? 1.0f : 0.0f, (h1 == t1) ? 1.0f : 0.0f), de);
        }
        if (WANT_GRAD) {
            const f32x2 kk = mul2(de, rinv[c]);
            t.fx[hf] = fma2(kk, dx[c], t.fx[hf]); t.fy[hf] = fma2(kk, dy[c], t.fy[hf]); t.fz[hf] = fma2(kk, dz[c], t.fz[hf]);
            gx[a] = fma2(kk, dx[c], gx[a]); gy[a] = fma2(kk, dy[c], gy[a]); gzz[a] = fma2(kk, dz[c], gzz[a]);
        }
    }
    if (WANT_GRAD) {
#pragma unroll
        for (int a = 0; a < NP; ++a) {
            const float sx = sum2(gx[a]), sy = sum2(gy[a]), sz = sum2(gzz[a]);
            if (PRE) {
                *reinterpret_cast<float2 *>(gxy + 2 * off[a]) = make_float2(pre[a].gx - sx, pre[a].gy - sy);
                *reinterpret_cast<float *>(gz + off[a]) = pre[a].gz - sz;
            } else {
                float2 g = *reinterpret_cast<float2 *>(gxy + 2 * off[a]);
                g.x -= sx; g.y -= sy;
                *reinterpret_cast<float2 *>(gxy + 2 * off[a]) = g;
                *reinterpret_cast<float *>(gz + off[a]) -= sz;
            }
        }
    }
}

template <int CLS, bool WANT_GRAD, bool SCHED_PARAM>
__device__ __forceinline__ void record_class(const DevParams &P, const TppLigand &L, int &pos, int n2, int n1, PairTile &t,
                                             PairAcc *acc,
                                             const char *xy, const char *zz, char *gxy, char *gz)
{
    if (n2 > 0) {
        // the partners of double record r+1 are read ahead of record r's arithmetic (measured +3 %, profiles/r1f.md:
        // the LDS latency is otherwise exposed at the top of every record); partners are distinct within a group,
        // so reading a force accumulator one record early is safe
        constexpr int STEP = 1 + 2 * (1 + CLS);
        PartnerRegs cur[2], nxt[2];
        {
            const uint4 h = tpp_quad<SCHED_PARAM>(L, pos);
            load_partner<WANT_GRAD>(h.x, xy, zz, gxy, gz, cur[0]);
            load_partner<WANT_GRAD>(h.y, xy, zz, gxy, gz, cur[1]);
        }
        for (int r = 0; r < n2; ++r) {
            nxt[0] = cur[0]; nxt[1] = cur[1];
            if (r + 1 < n2) {
                const uint4 h = tpp_quad<SCHED_PARAM>(L, pos + STEP);
                load_partner<WANT_GRAD>(h.x, xy, zz, gxy, gz, nxt[0]);
                load_partner<WANT_GRAD>(h.y, xy, zz, gxy, gz, nxt[1]);
            }
            record_block<2, CLS, WANT_GRAD, SCHED_PARAM, true>(P, L, pos, t, acc, xy, zz, gxy, gz, cur);
            cur[0] = nxt[0]; cur[1] = nxt[1];
        }
    }
    if (n1) record_block<1, CLS, WANT_GRAD, SCHED_PARAM>(P, L, pos, t, acc, xy, zz, gxy, gz);
}

// pose[k * ps] = k-th pose component of this thread; grad[k * gs] receives the k-th gradient component.
// `sm` = this warp's shared memory (tpp_warp_floats floats).  Returns E = e_grid + e_wall + e_intra.
template <bool WANT_GRAD, bool SCHED_PARAM, bool EQ4 = false>
__device__ __forceinline__ float eval_pose_thread(const DevParams &P, const DevGrid &G, const TppLigand &L,
                                                  const float *__restrict__ pose, int ps,
                                                  float *__restrict__ grad, int gs,
                                                  float *__restrict__ sm, EvalTerms &terms)
{
    const int lane = threadIdx.x & 31;
    const int N = L.N, T = L.T;
    const int rg = WANT_GRAD ? max(3 * N, 12 * T) : 12 * T;
    float2 *const xy = reinterpret_cast<float2 *>(sm) + lane;                      // [N]   stride 32
    float *const zz = sm + 64 * N + lane;                                          // [N]
    float *const rbase = sm + 96 * N;
    float2 *const fr = reinterpret_cast<float2 *>(rbase) + lane;                   // [T][6] frames of fragments 0..T-1 (phase 1 only)
    float2 *const gxy = reinterpret_cast<float2 *>(rbase) + lane;                  // [N]
    float *const gz = rbase + 64 * N + lane;                                       // [N]
    // force / torque sums of fragments 1..T: fragment f -> (Fx,Fy) (Fz,Mx) in fmA[2(f-1)], fmA[2(f-1)+1], My, Mz in fmB[..]
    float2 *const fmA = L.fm_alias ? gxy : reinterpret_cast<float2 *>(rbase + 32 * rg) + lane;   // [2T] stride 32
    float *const fmB = L.fm_alias ? gz : rbase + 32 * rg + 128 * T + lane;                       // [2T] stride 32

    const float tx = (pose[0] - G.rx) - G.rdx;
    const float ty = (pose[ps] - G.ry) - G.rdy;
    const float tz = (pose[2 * ps] - G.rz) - G.rdz;

    // ---- phase 1: A2 -------------------------------------------------------------------------------
    {
        // The torsion angles are fetched in one burst and parked in the z column: theta_k at slot N-T+k, which phase 1
        // writes only after fragment k+1 has consumed it (every later fragment owns at least one slot).  One exposed
        // global-load latency instead of one per fragment.
        for (int k = 0; k < T; ++k) zz[(N - T + k) * 32] = pose[(7 + k) * ps];
        Rot3 A = quat_to_rot(pose[3 * ps], pose[4 * ps], pose[5 * ps], pose[6 * ps]);
        float c0 = 0.0f, c1 = 0.0f, c2 = 0.0f;                                     // pivot-relative
        int s = 0;
        float sn_n = 0.0f, cs_n = 1.0f;                                            // sin / cos of the NEXT torsion (independent work
        if (T > 0) sincos_cw(zz[(N - T) * 32], sn_n, cs_n);                        // for the scheduler while a frame is composed)
        for (int f = 0; f <= T; ++f) {
            const float sn = sn_n, cs = cs_n;
            if (f < T && f > 0) sincos_cw(zz[(N - T + f) * 32], sn_n, cs_n);
            if (f > 0) {
                const int k = f - 1;
                const float4 u = L.tors_axis[k];
                const float4 b = L.tors_pt[k];
                const int p = __float_as_int(u.w);
                const float2 p0 = fr[(6 * p) * 32], p1 = fr[(6 * p + 1) * 32], p2 = fr[(6 * p + 2) * 32];
                const float2 p3 = fr[(6 * p + 3) * 32], p4 = fr[(6 * p + 4) * 32], p5 = fr[(6 * p + 5) * 32];
                const float omc = 1.0f - cs;
                const float ox = omc * u.x, oy = omc * u.y, oz = omc * u.z;
                const float sx = sn * u.x, sy = sn * u.y, sz = sn * u.z;
                const float r00 = fmaf(ox, u.x, cs), r01 = fmaf(ox, u.y, -sz), r02 = fmaf(ox, u.z, sy);
                const float r10 = fmaf(ox, u.y, sz), r11 = fmaf(oy, u.y, cs), r12 = fmaf(oy, u.z, -sx);
                const float r20 = fmaf(ox, u.z, -sy), r21 = fmaf(oy, u.z, sx), r22 = fmaf(oz, u.z, cs);
                // v = b - Rod b
                const float v0 = b.x - fmaf(r00, b.x, fmaf(r01, b.y, r02 * b.z));
                const float v1 = b.y - fmaf(r10, b.x, fmaf(r11, b.y, r12 * b.z));
                const float v2 = b.z - fmaf(r20, b.x, fmaf(r21, b.y, r22 * b.z));
                // parent frame: rows (p0.x p0.y p1.x) (p1.y p2.x p2.y) (p3.x p3.y p4.x), offset (p4.y p5.x p5.y)
                c0 = fmaf(p0.x, v0, fmaf(p0.y, v1, fmaf(p1.x, v2, p4.y)));
                c1 = fmaf(p1.y, v0, fmaf(p2.x, v1, fmaf(p2.y, v2, p5.x)));
                c2 = fmaf(p3.x, v0, fmaf(p3.y, v1, fmaf(p4.x, v2, p5.y)));
                A.m00 = fmaf(p0.x, r00, fmaf(p0.y, r10, p1.x * r20));
                A.m01 = fmaf(p0.x, r01, fmaf(p0.y, r11, p1.x * r21));
                A.m02 = fmaf(p0.x, r02, fmaf(p0.y, r12, p1.x * r22));
                A.m10 = fmaf(p1.y, r00, fmaf(p2.x, r10, p2.y * r20));
                A.m11 = fmaf(p1.y, r01, fmaf(p2.x, r11, p2.y * r21));
                A.m12 = fmaf(p1.y, r02, fmaf(p2.x, r12, p2.y * r22));
                A.m20 = fmaf(p3.x, r00, fmaf(p3.y, r10, p4.x * r20));
                A.m21 = fmaf(p3.x, r01, fmaf(p3.y, r11, p4.x * r21));
                A.m22 = fmaf(p3.x, r02, fmaf(p3.y, r12, p4.x * r22));
            }
            if (f < T) {                                                            // a later fragment may hang off this one
                fr[(6 * f) * 32] = make_float2(A.m00, A.m01);
                fr[(6 * f + 1) * 32] = make_float2(A.m02, A.m10);
                fr[(6 * f + 2) * 32] = make_float2(A.m11, A.m12);
                fr[(6 * f + 3) * 32] = make_float2(A.m20, A.m21);
                fr[(6 * f + 4) * 32] = make_float2(A.m22, c0);
                fr[(6 * f + 5) * 32] = make_float2(c1, c2);
            }
            const int s_end = L.frag_end[f];
            for (; s < s_end; ++s) {
                const float4 a = L.atom_ref[s];
                xy[s * 32] = make_float2(fmaf(A.m00, a.x, fmaf(A.m01, a.y, fmaf(A.m02, a.z, c0))),
                                         fmaf(A.m10, a.x, fmaf(A.m11, a.y, fmaf(A.m12, a.z, c1))));
                zz[s * 32] = fmaf(A.m20, a.x, fmaf(A.m21, a.y, fmaf(A.m22, a.z, c2)));
            }
        }
        if (WANT_GRAD)
            for (int i = 0; i < N; ++i) {                                           // the frames are dead: the region becomes the force array
                gxy[i * 32] = make_float2(0.0f, 0.0f);
                gz[i * 32] = 0.0f;
            }
    }

    // ---- phase 2: A3 + A4, one group per tile ----------------------------------------------------------
    float e_intra = 0.0f, e_grid = 0.0f, e_wall = 0.0f;
    {
        const char *xyb = reinterpret_cast<const char *>(xy), *zzb = reinterpret_cast<const char *>(zz);
        char *gxyb = reinterpret_cast<char *>(gxy), *gzb = reinterpret_cast<char *>(gz);
        const f32x2 z2 = bc2(0.0f);
        PairAcc acc[2] = {{z2, z2, z2, z2, z2}, {z2, z2, z2, z2, z2}};
        int pos = 0;
        for (int g = 0; g < L.n_groups; ++g) {
            const uint4 hdr = tpp_quad<SCHED_PARAM>(L, pos++);
            PairTile t;
            CellRef cr[TPP_TILE];
            float4 q0[TPP_TILE], q1[TPP_TILE];
            float ax[TPP_TILE], ay[TPP_TILE], az[TPP_TILE];
#pragma unroll
            for (int k = 0; k < TPP_TILE; ++k) {
                const int i = (int)((hdr.x >> (8 * k)) & 0xffu);
                const float2 a = xy[i * 32];
                ax[k] = a.x; ay[k] = a.y; az[k] = zz[i * 32];
                cr[k] = locate_cell(G, ax[k] + tx, ay[k] + ty, az[k] + tz);
                const Cell8 *e0 = G.packed + (size_t)__float_as_int(L.atom_ref[i].w) + cr[k].idx;
                ldg_cell(e0, q0[k], q1[k]);                                     // consumed after the records
            }
#pragma unroll
            for (int hf = 0; hf < 2; ++hf) {
                t.x[hf] = pk2(ax[2 * hf], ax[2 * hf + 1]); t.y[hf] = pk2(ay[2 * hf], ay[2 * hf + 1]); t.z[hf] = pk2(az[2 * hf], az[2 * hf + 1]);
                t.fx[hf] = t.fy[hf] = t.fz[hf] = z2;
            }
            record_class<0, WANT_GRAD, SCHED_PARAM>(P, L, pos, (int)(hdr.y & 0xffu), (int)((hdr.y >> 8) & 0xffu), t, acc, xyb, zzb, gxyb, gzb);
            record_class<1, WANT_GRAD, SCHED_PARAM>(P, L, pos, (int)((hdr.y >> 16) & 0xffu), (int)(hdr.y >> 24), t, acc, xyb, zzb, gxyb, gzb);
            record_class<2, WANT_GRAD, SCHED_PARAM>(P, L, pos, (int)(hdr.z & 0xffu), (int)((hdr.z >> 8) & 0xffu), t, acc, xyb, zzb, gxyb, gzb);
            const int n_live = (int)(hdr.z >> 16);
            float tfx[TPP_TILE], tfy[TPP_TILE], tfz[TPP_TILE];
#pragma unroll
            for (int hf = 0; hf < 2; ++hf) {
                up2(t.fx[hf], tfx[2 * hf], tfx[2 * hf + 1]); up2(t.fy[hf], tfy[2 * hf], tfy[2 * hf + 1]); up2(t.fz[hf], tfz[2 * hf], tfz[2 * hf + 1]);
            }
#pragma unroll
            for (int k = 0; k < TPP_TILE; ++k) {
                if (k < n_live) {                                               // padding slots of the last tile: skipped
                    float gx, gy, gz_;
                    if (EQ4 && WANT_GRAD) {                                     // NEXT-2: eq. 4, three more cells per atom (not prefetched)
                        const int ia = (int)((hdr.x >> (8 * k)) & 0xffu);
                        const Cell8 *cell = G.packed + (size_t)__float_as_int(L.atom_ref[ia].w) + cr[k].idx;
                        e_grid += trilinear_eq4(G, cr[k], cell, q0[k], q1[k], e_wall, gx, gy, gz_);
                    } else
                        e_grid += trilinear(G, cr[k], q0[k], q1[k], e_wall, gx, gy, gz_);
                    if (WANT_GRAD) {
                        const int i = (int)((hdr.x >> (8 * k)) & 0xffu);
                        float2 gi = gxy[i * 32];
                        gi.x += fmaf(P.sigma, gx, tfx[k]);
                        gi.y += fmaf(P.sigma, gy, tfy[k]);
                        gxy[i * 32] = gi;
                        gz[i * 32] += fmaf(P.sigma, gz_, tfz[k]);
                    }
                }
            }
        }
        const float a = sum2(add2(acc[0].a, acc[1].a)), b = sum2(add2(acc[0].b, acc[1].b)), rep = sum2(add2(acc[0].rep, acc[1].rep));
        const float hyd = sum2(add2(acc[0].hyd, acc[1].hyd)), hb = sum2(add2(acc[0].hb, acc[1].hb));
        e_intra = fmaf(P.eA, a, fmaf(P.eB, b, P.sigma * fmaf(0.5f, rep, fmaf(-0.7f, hb, -hyd))));
    }

    // ---- phases 3 + 4: A5 (sigma-scaled until the stores) ------------------------------------------------
    if (WANT_GRAD) {
        float rFx = 0.f, rFy = 0.f, rFz = 0.f, rMx = 0.f, rMy = 0.f, rMz = 0.f;   // root fragment, about the pivot
        int s = 0;
        for (int f = 0; f <= T; ++f) {
            float ox = 0.0f, oy = 0.0f, oz = 0.0f;                                // origin of the fragment, pivot-relative
            if (f > 0) {
                const int bs = L.tors_b[f - 1];
                const float2 ob = xy[bs * 32];
                ox = ob.x; oy = ob.y; oz = zz[bs * 32];
            }
            float Fx = 0.f, Fy = 0.f, Fz = 0.f, Mx = 0.f, My = 0.f, Mz = 0.f;
            const int s_end = L.frag_end[f];
            for (; s < s_end; ++s) {
                const float2 v = xy[s * 32], gp = gxy[s * 32];
                const float gz_ = gz[s * 32];
                const float lx = v.x - ox, ly = v.y - oy, lz = zz[s * 32] - oz;
                Fx += gp.x; Fy += gp.y; Fz += gz_;
                Mx = fmaf(ly, gz_, fmaf(-lz, gp.y, Mx));
                My = fmaf(lz, gp.x, fmaf(-lx, gz_, My));
                Mz = fmaf(lx, gp.y, fmaf(-ly, gp.x, Mz));
            }
            if (f == 0) { rFx = Fx; rFy = Fy; rFz = Fz; rMx = Mx; rMy = My; rMz = Mz; }
            else {
                fmA[(2 * (f - 1)) * 32] = make_float2(Fx, Fy);
                fmA[(2 * (f - 1) + 1) * 32] = make_float2(Fz, Mx);
                fmB[(2 * (f - 1)) * 32] = My;
                fmB[(2 * (f - 1) + 1) * 32] = Mz;
            }
        }
        for (int f = T; f >= 1; --f) {
            const float2 a0 = fmA[(2 * (f - 1)) * 32], a1 = fmA[(2 * (f - 1) + 1) * 32];
            const float Fx = a0.x, Fy = a0.y, Fz = a1.x, Mx = a1.y, My = fmB[(2 * (f - 1)) * 32], Mz = fmB[(2 * (f - 1) + 1) * 32];
            const int as = L.tors_a[f - 1], bs = L.tors_b[f - 1];
            const float4 tp = L.tors_pt[f - 1];
            const float2 xb = xy[bs * 32], xa = xy[as * 32];
            const float zb = zz[bs * 32], za = zz[as * 32];
            const float w = tp.w * P.sigma;                                     // 1/|b - a|, and the sign of the scaled forces
            const float ux = (xb.x - xa.x) * w, uy = (xb.y - xa.y) * w, uz = (zb - za) * w;   // lab-frame unit axis (x sigma)
            grad[(6 + f - 1) * gs] = fmaf(ux, Mx, fmaf(uy, My, uz * Mz));
            const int p = __float_as_int(L.tors_axis[f - 1].w);                 // parent fragment
            if (p > 0) {                                                        // uniform
                const int pb = L.tors_b[p - 1];
                const float2 o = xy[pb * 32];
                const float lx = xb.x - o.x, ly = xb.y - o.y, lz = zb - zz[pb * 32];
                float2 b0 = fmA[(2 * (p - 1)) * 32], b1 = fmA[(2 * (p - 1) + 1) * 32];
                b0.x += Fx; b0.y += Fy; b1.x += Fz;
                b1.y += Mx + fmaf(ly, Fz, -lz * Fy);
                fmA[(2 * (p - 1)) * 32] = b0; fmA[(2 * (p - 1) + 1) * 32] = b1;
                fmB[(2 * (p - 1)) * 32] += My + fmaf(lz, Fx, -lx * Fz);
                fmB[(2 * (p - 1) + 1) * 32] += Mz + fmaf(lx, Fy, -ly * Fx);
            } else {
                rFx += Fx; rFy += Fy; rFz += Fz;
                rMx += Mx + fmaf(xb.y, Fz, -zb * Fy);
                rMy += My + fmaf(zb, Fx, -xb.x * Fz);
                rMz += Mz + fmaf(xb.x, Fy, -xb.y * Fx);
            }
        }
        grad[0] = P.sigma * rFx; grad[gs] = P.sigma * rFy; grad[2 * gs] = P.sigma * rFz;
        grad[3 * gs] = P.sigma * rMx; grad[4 * gs] = P.sigma * rMy; grad[5 * gs] = P.sigma * rMz;
    }
    terms.e_grid = e_grid; terms.e_wall = e_wall; terms.e_intra = e_intra;
    return e_grid + e_wall + e_intra;
}
