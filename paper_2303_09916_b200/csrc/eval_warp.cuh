// eval_warp.cuh -- fused pose -> coordinates -> energy + gradient, ONE WARP PER POSE (SURVEY.md 8(a)
// A2-A5).  The latency evaluator behind the search kernels, where a few hundred copies must fill the
// GPU and each copy's evaluations are sequential (the throughput evaluator is eval_thread.cuh).
//
//   A2 kinematics : every lane owns atoms i = lane, lane+32, ... and walks the torsions on the path
//                   from the atom's fragment to the root (deepest first), one Rodrigues rotation
//                   about the reference-frame axis each, then x = t + R(q) y (box-relative).
//   A3 inter term : one 32-byte gather (the cell's 8 corners) from the packed map of the atom's type, trilinear energy
//                   (eq. 2, 198-207) and the partial derivatives of the interpolant (eq. 3,
//                   213-219); clamp + quadratic wall outside the box.
//   A4 intra term : host-built conflict-free schedule, 32 pairs per round; forces go to the per-warp
//                   shared-memory gradient array with plain read-modify-writes in two phases
//                   (all sources, then all destinations) -> deterministic, no float atomics.
//   A5 chain rule : force = sum g_i, torque = sum (x_i - t) x g_i, dE/dtheta_k = u_k . sum_{subtree} (x_i - x_b) x g_i.
//
// All lanes of the warp return the same energy.  `pose` (7+T floats) and `grad` (6+T floats) live
// in shared memory owned by the warp; `scratch` is eval_scratch_floats() floats of the same.
#pragma once

#include "common.cuh"
#include "eval_thread.cuh"   // EvalTerms
#include "mathx.cuh"

// A2 for atom i: box-relative position.  `sn`, `cs` hold sin/cos(theta_k).
__device__ __forceinline__ void atom_coords(const DevLigand &L, const Rot3 &R, float tx, float ty, float tz,
                                            const float *sn, const float *cs, int i,
                                            float &x0, float &x1, float &x2, int &map_off)
{
    const float4 a = __ldg(&L.atom_ref[i]);
    float y0 = a.x, y1 = a.y, y2 = a.z;
    map_off = __float_as_int(a.w);
    int f = __ldg(&L.atom_topo[i]).x;
    while (f > 0) {
        const int k = f - 1;
        const float4 u = __ldg(&L.tors_axis[k]);
        const float4 b = __ldg(&L.tors_pt[k]);
        const float c = cs[k];
        rodrigues(u.x, u.y, u.z, b.x, b.y, b.z, sn[k], c, 1.0f - c, y0, y1, y2);
        f = __float_as_int(b.w);
    }
    x0 = fmaf(R.m00, y0, fmaf(R.m01, y1, fmaf(R.m02, y2, tx)));
    x1 = fmaf(R.m10, y0, fmaf(R.m11, y1, fmaf(R.m12, y2, ty)));
    x2 = fmaf(R.m20, y0, fmaf(R.m21, y1, fmaf(R.m22, y2, tz)));
}

// Coordinates only (used by the top-k kernel): xs[c*np + i].
__device__ __forceinline__ void pose_coords_warp(const DevLigand &L, const float *pose, float *xs, float *sc)
{
    const int lane = threadIdx.x & 31, T = L.T, np = L.n_pad;
    float *sn = sc, *cs = sc + ((T + 3) & ~3);
    if (lane < T) {
        float s, c;
        sincos_cw(pose[7 + lane], s, c);
        sn[lane] = s; cs[lane] = c;
    }
    const Rot3 R = quat_to_rot(pose[3], pose[4], pose[5], pose[6]);
    __syncwarp();
    for (int i = lane; i < L.N; i += 32) {
        float x0, x1, x2;
        int mo;
        atom_coords(L, R, pose[0], pose[1], pose[2], sn, cs, i, x0, x1, x2, mo);
        xs[i] = x0; xs[np + i] = x1; xs[2 * np + i] = x2;
    }
    __syncwarp();
}

// Per-atom 3-vectors of the warp evaluator in shared memory, two layouts chosen per launch (search.cu):
//   VEC4 : float4 per atom -- one 16-byte access instead of three 4-byte ones: fewer instructions on the single
//          dependent chain of a latency-bound launch (few hundred copies), but random atom indices then collide in the
//          8 bank groups of a quarter-warp phase (about 3x the shared-memory wavefronts);
//   !VEC4: three rows [c * n_pad + i] -- conflict-free for N <= 32 and nearly so above; right for throughput-bound
//          launches with large ligands (configs[4]: 75.6 vs 60.7 M evals/s, profiles/r1l.md).
template <bool VEC4>
__device__ __forceinline__ void ld3(const float *base, int np, int i, float &x, float &y, float &z)
{
    if (VEC4) { const float4 v = reinterpret_cast<const float4 *>(base)[i]; x = v.x; y = v.y; z = v.z; }
    else { x = base[i]; y = base[np + i]; z = base[2 * np + i]; }
}
template <bool VEC4>
__device__ __forceinline__ void st3(float *base, int np, int i, float x, float y, float z)
{
    if (VEC4) reinterpret_cast<float4 *>(base)[i] = make_float4(x, y, z, 0.0f);
    else { base[i] = x; base[np + i] = y; base[2 * np + i] = z; }
}

template <bool WANT_GRAD, bool EQ4 = false, bool VEC4 = true>
__device__ __forceinline__ float eval_pose_warp(const DevParams &P, const DevGrid &G, const DevLigand &L,
                                             const float *pose, float *grad, float *scratch, EvalTerms *terms)
{
    const int lane = threadIdx.x & 31;
    const int N = L.N, T = L.T, np = L.n_pad;
    float *xs = scratch, *gs = scratch + 4 * np;                                 // layouts: ld3 / st3 above
    float *sn = scratch + 8 * np, *cs = sn + ((T + 3) & ~3);

    if (lane < T) {
        float s, c;
        sincos_cw(pose[7 + lane], s, c);
        sn[lane] = s; cs[lane] = c;
    }
    const float tx = (pose[0] - G.rx) - G.rdx, ty = (pose[1] - G.ry) - G.rdy, tz = (pose[2] - G.rz) - G.rdz;
    const Rot3 R = quat_to_rot(pose[3], pose[4], pose[5], pose[6]);
    __syncwarp();

    // ---- A2 + A3 -------------------------------------------------------------------------------
    float e_grid = 0.0f, e_wall = 0.0f;
    for (int i = lane; i < N; i += 32) {
        float x0, x1, x2, gx, gy, gz;
        int map_off;
        atom_coords(L, R, tx, ty, tz, sn, cs, i, x0, x1, x2, map_off);
        st3<VEC4>(xs, np, i, x0, x1, x2);
        const CellRef cr = locate_cell(G, x0, x1, x2);
        float4 q0, q1;
        const Cell8 *cell = G.packed + (size_t)map_off + cr.idx;
        ldg_cell(cell, q0, q1);
        if (EQ4 && WANT_GRAD) e_grid += trilinear_eq4(G, cr, cell, q0, q1, e_wall, gx, gy, gz);   // NEXT-2: eq. 4 gradient
        else e_grid += trilinear(G, cr, q0, q1, e_wall, gx, gy, gz);
        if (WANT_GRAD) st3<VEC4>(gs, np, i, gx, gy, gz);
    }
    __syncwarp();

    // ---- A4 ------------------------------------------------------------------------------------
    // Branch-free rounds: an idle lane or an out-of-range pair gets the surface distance 1e18, for which every
    // term and derivative is exactly 0 (weights folded into the exponents as in eval_thread.cuh, see DevParams);
    // the next round's record is fetched while this one computes.
    float aA = 0.0f, aB = 0.0f, aRep = 0.0f, aHyd = 0.0f, aHb = 0.0f;
    {
        const float4 *sched = reinterpret_cast<const float4 *>(L.sched) + lane;
        const int n_rounds = L.n_rounds;
        float4 raw = n_rounds > 0 ? __ldg(sched) : make_float4(0.f, 0.f, 0.f, 0.f);
        for (int r = 0; r < n_rounds; ++r) {
            const float4 cur = raw;
            if (r + 1 < n_rounds) raw = __ldg(sched + (r + 1) * 32);
            const int ij = __float_as_int(cur.x);
            const bool valid = ij >= 0;
            const int i = valid ? (ij & 0xffff) : 0, j = valid ? (ij >> 16) : 0;
            float xi, yi, zi, xj, yj, zj;
            ld3<VEC4>(xs, np, i, xi, yi, zi);
            ld3<VEC4>(xs, np, j, xj, yj, zj);
            const float dx = xi - xj, dy = yi - yj, dz = zi - zj;
            const float r2 = fmaf(dz, dz, fmaf(dy, dy, fmaf(dx, dx, 1e-12f)));
            const float rinv = fast_rsqrt(r2);
            const float d = (valid && r2 < P.cutoff2) ? fmaf(r2, rinv, -cur.y) : 1.0e18f;
            const float A = fast_ex2(fmaf(d * -5.770780163555854f, d, P.lw1));
            const float B = fast_ex2(fmaf(d, fmaf(d, -0.36067376022224085f, 2.1640425613334453f), P.lw2 - 3.2460638420001677f));
            const float m = fminf(d, 0.0f);
            const float c4m = P.c4 * m;
            aA += A; aB += B;
            aRep = fmaf(c4m, m, aRep);
            float de = fmaf(d, fmaf(P.q, B, A), fmaf(P.m3q, B, c4m));            // sigma dE/dd
            const float th = 1.5f - d, hh = __saturatef(th);
            aHyd = fmaf(cur.z, hh, aHyd);
            de = fmaf(cur.z, (hh == th) ? 1.0f : 0.0f, de);
            const float tb = d * -1.4285714285714286f, hb = __saturatef(tb);
            aHb = fmaf(cur.w, hb, aHb);
            de = fmaf(cur.w, (hb == tb) ? 1.0f : 0.0f, de);
            if (WANT_GRAD) {
                const float k = P.sigma * de * rinv;
                const float fx = k * dx, fy = k * dy, fz = k * dz;
                if (valid) {                                                  // loads before stores (the rows may alias for the compiler)
                    float a0, a1, a2;
                    ld3<VEC4>(gs, np, i, a0, a1, a2);
                    st3<VEC4>(gs, np, i, a0 + fx, a1 + fy, a2 + fz);
                }
                __syncwarp();
                if (valid) {
                    float a0, a1, a2;
                    ld3<VEC4>(gs, np, j, a0, a1, a2);
                    st3<VEC4>(gs, np, j, a0 - fx, a1 - fy, a2 - fz);
                }
                __syncwarp();
            }
        }
    }
    float e_intra = fmaf(P.eA, aA, fmaf(P.eB, aB, P.sigma * fmaf(0.5f, aRep, fmaf(-0.7f, aHb, -aHyd))));

    // the lanes' partial energies are added in double: the total feeds the Armijo and Metropolis decisions, and a
    // 32-term fp32 tree would add ~1e-6 |E| of noise to differences the line search has to resolve
    float e_total;
    if (terms) {
        const double dg = warp_sum_d((double)e_grid), dw = warp_sum_d((double)e_wall), di = warp_sum_d((double)e_intra);
        terms->e_grid = (float)dg; terms->e_wall = (float)dw; terms->e_intra = (float)di;
        e_total = (float)(dg + dw + di);
    } else
        e_total = (float)warp_sum_d((double)e_grid + (double)e_wall + (double)e_intra);

    // ---- A5 ------------------------------------------------------------------------------------
    // With p_i = x_i - t (lever arm about the pivot) and m_i = p_i x g_i:
    //   torque = sum m_i;   dE/dtheta_k = u_k . sum_{i in subtree k} m_i - (u_k x p_b) . sum_{i in subtree k} g_i.
    // Lane k prepares (u_k, u_k x p_b); every lane then forms its atoms' share of all T torsion sums in its own
    // column tsum[k][lane], and lane k adds row k -- no per-torsion shuffle reductions.
    if (WANT_GRAD) {
        float *tsum = cs + ((T + 3) & ~3);                                       // [T][32]
        float4 *uw = reinterpret_cast<float4 *>(tsum + 32 * T);                  // [T][2]
        for (int k = lane; k < T; k += 32) {
            const int2 ab = __ldg(&L.tors_ab[k]);
            float bx, by, bz, ax, ay, az;
            ld3<VEC4>(xs, np, ab.y, bx, by, bz);
            ld3<VEC4>(xs, np, ab.x, ax, ay, az);
            float ux = bx - ax, uy = by - ay, uz = bz - az;
            const float inv = 1.0f / sqrtf(ux * ux + uy * uy + uz * uz);
            ux *= inv; uy *= inv; uz *= inv;
            const float lx = bx - tx, ly = by - ty, lz = bz - tz;
            uw[2 * k] = make_float4(ux, uy, uz, 0.0f);
            uw[2 * k + 1] = make_float4(uy * lz - uz * ly, uz * lx - ux * lz, ux * ly - uy * lx, 0.0f);
        }
        for (int k = 0; k < T; ++k) tsum[k * 32 + lane] = 0.0f;
        __syncwarp();
        float fx = 0.f, fy = 0.f, fz = 0.f, qx = 0.f, qy = 0.f, qz = 0.f;
        for (int i = lane; i < N; i += 32) {
            float gx, gy, gz, px, py, pz;
            ld3<VEC4>(gs, np, i, gx, gy, gz);
            ld3<VEC4>(xs, np, i, px, py, pz);
            px -= tx; py -= ty; pz -= tz;
            const float mx = py * gz - pz * gy, my = pz * gx - px * gz, mz = px * gy - py * gx;
            fx += gx; fy += gy; fz += gz;
            qx += mx; qy += my; qz += mz;
            unsigned mask = (unsigned)__ldg(&L.atom_topo[i]).y;
            while (mask) {                                                        // torsions on the path to the root
                const int k = __ffs(mask) - 1;
                mask &= mask - 1;
                const float4 u = uw[2 * k], w = uw[2 * k + 1];
                tsum[k * 32 + lane] += fmaf(u.x, mx, fmaf(u.y, my, u.z * mz)) - fmaf(w.x, gx, fmaf(w.y, gy, w.z * gz));
            }
        }
        __syncwarp();
        fx = warp_sum(fx); fy = warp_sum(fy); fz = warp_sum(fz);
        qx = warp_sum(qx); qy = warp_sum(qy); qz = warp_sum(qz);
        if (lane == 0) {
            grad[0] = fx; grad[1] = fy; grad[2] = fz;
            grad[3] = qx; grad[4] = qy; grad[5] = qz;
        }
        for (int k = lane; k < T; k += 32) {
            float c0 = 0.f, c1 = 0.f, c2 = 0.f, c3 = 0.f;
#pragma unroll
            for (int l = 0; l < 32; l += 4) {
                const int a = (l + lane) & 31;                                    // skewed: conflict-free
                c0 += tsum[k * 32 + a]; c1 += tsum[k * 32 + ((a + 1) & 31)];
                c2 += tsum[k * 32 + ((a + 2) & 31)]; c3 += tsum[k * 32 + ((a + 3) & 31)];
            }
            grad[6 + k] = (c0 + c1) + (c2 + c3);
        }
        __syncwarp();
    }
    return e_total;
}
