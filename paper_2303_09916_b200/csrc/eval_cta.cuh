// eval_cta.cuh -- fused pose -> coordinates -> energy + gradient, ONE CTA OF FOUR WARPS PER POSE.
//
// The latency form of eval_warp.cuh for the Barzilai-Borwein search ("only needs a vector inner product ...
// and does not need to perform line search"): BB makes ONE evaluation per iteration, so the four warps of the CTA search
// kernel have no line-search trials to speculate on -- they share the evaluation instead.  Atoms are spread over the 128
// threads, and the conflict-free pair rounds over the warps (round r goes to warp r mod 4): a 32-atom, 355-pair ligand
// runs 4 rounds per warp instead of 14.  Every warp accumulates its pair forces in its OWN force array (no inter-warp
// read-modify-write); the arrays are added before the chain rule, which warp 0 carries out exactly as eval_pose_warp.
// Same arithmetic per atom, pair and torsion as eval_pose_warp; the force and energy sums are taken in another order,
// so the results agree to round-off, not bit for bit.
//
// Every thread of the CTA must call it with the same pose values; `pose` may be per-warp copies.  All threads return the
// same energy; the gradient goes to `grad` (shared memory).  scratch0 = the scratch of warp 0 (eval_scratch_floats()),
// sc_stride = distance between the warps' scratch areas; esum = 4 doubles of shared memory.
#pragma once

#include "eval_warp.cuh"

template <bool EQ4, bool VEC4>
__device__ __forceinline__ float eval_pose_cta(const DevParams &P, const DevGrid &G, const DevLigand &L,
                                               const float *pose, float *grad, float *scratch0, int sc_stride, double *esum)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, tid = threadIdx.x;
    const int N = L.N, T = L.T, np = L.n_pad;
    float *const xs = scratch0;                                               // coordinates: warp 0's array, read by all
    float *const gs0 = scratch0 + 4 * np;                                     // warp 0's force array (grid forces + its pair rounds)
    float *const gsw = scratch0 + (size_t)warp * sc_stride + 4 * np;          // this warp's force array
    float *const sn = scratch0 + (size_t)warp * sc_stride + 8 * np, *const cs = sn + ((T + 3) & ~3);   // per warp (redundant)

    if (lane < T) {
        float s, c;
        sincos_cw(pose[7 + lane], s, c);
        sn[lane] = s; cs[lane] = c;
    }
    const float tx = (pose[0] - G.rx) - G.rdx, ty = (pose[1] - G.ry) - G.rdy, tz = (pose[2] - G.rz) - G.rdz;
    const Rot3 R = quat_to_rot(pose[3], pose[4], pose[5], pose[6]);
    if (warp > 0)
        for (int k = lane; k < 4 * np; k += 32) gsw[k] = 0.0f;
    __syncwarp();

    // ---- A2 + A3: one atom per thread ----
    float e_part = 0.0f, e_wall = 0.0f;
    for (int i = tid; i < N; i += 4 * 32) {
        float x0, x1, x2, gx, gy, gz;
        int map_off;
        atom_coords(L, R, tx, ty, tz, sn, cs, i, x0, x1, x2, map_off);
        st3<VEC4>(xs, np, i, x0, x1, x2);
        const CellRef cr = locate_cell(G, x0, x1, x2);
        float4 q0, q1;
        const Cell8 *cell = G.packed + (size_t)map_off + cr.idx;
        ldg_cell(cell, q0, q1);
        if (EQ4) e_part += trilinear_eq4(G, cr, cell, q0, q1, e_wall, gx, gy, gz);
        else e_part += trilinear(G, cr, q0, q1, e_wall, gx, gy, gz);
        st3<VEC4>(gs0, np, i, gx, gy, gz);
    }
    __syncthreads();

    // ---- A4: round r -> warp r mod 4 ----
    float aA = 0.0f, aB = 0.0f, aRep = 0.0f, aHyd = 0.0f, aHb = 0.0f;
    {
        const float4 *sched = reinterpret_cast<const float4 *>(L.sched) + lane;
        const int n_rounds = L.n_rounds;
        float4 raw = warp < n_rounds ? __ldg(sched + warp * 32) : make_float4(0.f, 0.f, 0.f, 0.f);
        for (int r = warp; r < n_rounds; r += 4) {
            const float4 cur = raw;
            if (r + 4 < n_rounds) raw = __ldg(sched + (r + 4) * 32);
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
            const float k = P.sigma * de * rinv;
            const float fx = k * dx, fy = k * dy, fz = k * dz;
            if (valid) {
                float a0, a1, a2;
                ld3<VEC4>(gsw, np, i, a0, a1, a2);
                st3<VEC4>(gsw, np, i, a0 + fx, a1 + fy, a2 + fz);
            }
            __syncwarp();
            if (valid) {
                float a0, a1, a2;
                ld3<VEC4>(gsw, np, j, a0, a1, a2);
                st3<VEC4>(gsw, np, j, a0 - fx, a1 - fy, a2 - fz);
            }
            __syncwarp();
        }
    }
    const float e_intra = fmaf(P.eA, aA, fmaf(P.eB, aB, P.sigma * fmaf(0.5f, aRep, fmaf(-0.7f, aHb, -aHyd))));
    const double ew = warp_sum_d((double)e_part + (double)e_wall + (double)e_intra);
    if (lane == 0) esum[warp] = ew;
    __syncthreads();
    const float e_total = (float)(((esum[0] + esum[1]) + esum[2]) + esum[3]);

    // ---- forces of the four warps added into warp 0's array ----
    for (int i = tid; i < N; i += 4 * 32) {
        float g0, g1, g2;
        ld3<VEC4>(gs0, np, i, g0, g1, g2);
#pragma unroll
        for (int w = 1; w < 4; ++w) {
            float h0, h1, h2;
            ld3<VEC4>(scratch0 + (size_t)w * sc_stride + 4 * np, np, i, h0, h1, h2);
            g0 += h0; g1 += h1; g2 += h2;
        }
        st3<VEC4>(gs0, np, i, g0, g1, g2);
    }
    __syncthreads();

    // ---- A5 by warp 0, as in eval_pose_warp ----
    if (warp == 0) {
        float *const sn0 = scratch0 + 8 * np, *const cs0 = sn0 + ((T + 3) & ~3);
        float *tsum = cs0 + ((T + 3) & ~3);                                      // [T][32]
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
            ld3<VEC4>(gs0, np, i, gx, gy, gz);
            ld3<VEC4>(xs, np, i, px, py, pz);
            px -= tx; py -= ty; pz -= tz;
            const float mx = py * gz - pz * gy, my = pz * gx - px * gz, mz = px * gy - py * gx;
            fx += gx; fy += gy; fz += gz;
            qx += mx; qy += my; qz += mz;
            unsigned mask = (unsigned)__ldg(&L.atom_topo[i]).y;
            while (mask) {
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
                const int a = (l + lane) & 31;
                c0 += tsum[k * 32 + a]; c1 += tsum[k * 32 + ((a + 1) & 31)];
                c2 += tsum[k * 32 + ((a + 2) & 31)]; c3 += tsum[k * 32 + ((a + 3) & 31)];
            }
            grad[6 + k] = (c0 + c1) + (c2 + c3);
        }
    }
    __syncthreads();
    return e_total;
}
