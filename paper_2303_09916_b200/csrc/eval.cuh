// eval.cuh -- fused pose -> coordinates -> energy + gradient, one warp per pose.
//
//   A2 kinematics : every lane owns atoms i = lane, lane+32, ... and walks the torsions on the path
//                   from the atom's fragment to the root (deepest first), one Rodrigues rotation
//                   about the reference-frame axis each, then x = t + R(q) y.
//   A3 inter term : 8 corner loads of the atom's type map, trilinear energy (eq. 2, 198-207)
//                   and the partial derivatives of the interpolant (eq. 3, 213-219); clamp + quadratic
//                   wall outside the box.
//   A4 intra term : host-built conflict-free schedule, 32 pairs per round; forces go to the per-warp
//                   shared-memory gradient array with plain read-modify-writes in two phases
//                   (all sources, then all destinations) -> deterministic, no float atomics.
//   A5 chain rule : force = sum g_i, torque = sum (x_i - t) x g_i, dE/dtheta_k = u_k . sum_{subtree} (x_i - x_b) x g_i.
//
// All lanes of the warp return the same energy.  `pose` (7+T floats) and `grad` (6+T floats) live
// in shared memory owned by the warp; `scratch` is eval_scratch_floats() floats of the same.
#pragma once

#include "common.cuh"

struct EvalTerms {
    float e_grid, e_wall, e_intra;
};

// Vina-style pair term on the surface distance d = r - (R_i + R_j).
// Returns e; dedr_over_r = (de/dr)/r so that the force on i is dedr_over_r * (x_i - x_j).
__device__ __forceinline__ float pair_term(const DevParams &P, float r2, float rsum, float wh, float whb,
                                           float &dedr_over_r)
{
    r2 = fmaxf(r2, 1e-12f);
    const float rinv = fast_rsqrt(r2);
    const float r = r2 * rinv;
    const float d = r - rsum;
    const float g1 = fast_ex2(-5.770780163555854f * d * d);          // exp(-(d/0.5)^2)
    const float dm3 = d - 3.0f;
    const float g2 = fast_ex2(-0.36067376022224085f * dm3 * dm3);    // exp(-((d-3)/2)^2)
    const float rep = fminf(d, 0.0f);
    const float hyd = __saturatef(1.5f - d);                         // 1 | 1.5-d | 0
    const float hb = __saturatef(d * -1.4285714285714286f);          // 1 | -d/0.7 | 0
    const float hyd_d = (d >= 0.5f && d < 1.5f) ? -1.0f : 0.0f;
    const float hb_d = (d >= -0.7f && d < 0.0f) ? -1.4285714285714286f : 0.0f;
    const float w1g1 = P.w[0] * g1, w2g2 = P.w[1] * g2, w3rep = P.w[2] * rep;
    float e = w1g1 + w2g2;
    e = fmaf(w3rep, rep, e);
    e = fmaf(wh, hyd, e);
    e = fmaf(whb, hb, e);
    float de = -8.0f * d * w1g1;
    de = fmaf(-0.5f * dm3, w2g2, de);
    de = fmaf(2.0f, w3rep, de);
    de = fmaf(wh, hyd_d, de);
    de = fmaf(whb, hb_d, de);
    dedr_over_r = de * rinv;
    return e;
}

// Trilinear energy and gradient of one atom + wall.  Returns e_grid; adds to e_wall; writes g.
__device__ __forceinline__ float atom_inter(const DevParams &P, const DevGrid &G, int map_off,
                                            float x, float y, float z, float &e_wall,
                                            float &gx, float &gy, float &gz)
{
    const float ovx = fminf(x - G.ox, 0.0f) + fmaxf(x - G.hx, 0.0f);
    const float ovy = fminf(y - G.oy, 0.0f) + fmaxf(y - G.hy, 0.0f);
    const float ovz = fminf(z - G.oz, 0.0f) + fmaxf(z - G.hz, 0.0f);
    const float ux = fminf(fmaxf((x - G.ox) * G.inv_h, 0.0f), (float)(G.nx - 1));
    const float uy = fminf(fmaxf((y - G.oy) * G.inv_h, 0.0f), (float)(G.ny - 1));
    const float uz = fminf(fmaxf((z - G.oz) * G.inv_h, 0.0f), (float)(G.nz - 1));
    const int ix = min((int)ux, G.nx - 2), iy = min((int)uy, G.ny - 2), iz = min((int)uz, G.nz - 2);
    const float px = ux - (float)ix, py = uy - (float)iy, pz = uz - (float)iz;
    const float *g0 = G.data + map_off + ((size_t)iz * G.ny + iy) * G.nx + ix;
    const size_t sy = G.nx, sz = (size_t)G.nx * G.ny;
    const float v000 = __ldg(g0), v100 = __ldg(g0 + 1);
    const float v010 = __ldg(g0 + sy), v110 = __ldg(g0 + sy + 1);
    const float v001 = __ldg(g0 + sz), v101 = __ldg(g0 + sz + 1);
    const float v011 = __ldg(g0 + sz + sy), v111 = __ldg(g0 + sz + sy + 1);
    // x-differences and x-interpolants on the four cell edges along x
    const float d00 = v100 - v000, d10 = v110 - v010, d01 = v101 - v001, d11 = v111 - v011;
    const float c00 = fmaf(px, d00, v000), c10 = fmaf(px, d10, v010);
    const float c01 = fmaf(px, d01, v001), c11 = fmaf(px, d11, v011);
    const float c0 = fmaf(py, c10 - c00, c00), c1 = fmaf(py, c11 - c01, c01);
    const float e = fmaf(pz, c1 - c0, c0);                                            // eq. 2
    const float dx0 = fmaf(py, d10 - d00, d00), dx1 = fmaf(py, d11 - d01, d01);
    float ggx = fmaf(pz, dx1 - dx0, dx0) * G.inv_h;                                   // eq. 3, x
    const float dy0 = c10 - c00, dy1 = c11 - c01;
    float ggy = fmaf(pz, dy1 - dy0, dy0) * G.inv_h;                                   // eq. 3, y
    float ggz = (c1 - c0) * G.inv_h;                                                  // eq. 3, z
    // clamped axes: lookup is constant there; quadratic wall k*overshoot^2
    if (ovx != 0.0f) ggx = 0.0f;
    if (ovy != 0.0f) ggy = 0.0f;
    if (ovz != 0.0f) ggz = 0.0f;
    const float k2 = 2.0f * P.k_wall;
    gx = fmaf(k2, ovx, ggx);
    gy = fmaf(k2, ovy, ggy);
    gz = fmaf(k2, ovz, ggz);
    e_wall += P.k_wall * (ovx * ovx + ovy * ovy + ovz * ovz);
    return e;
}

struct Rot3 {
    float m[9];
};

// q = (w,x,y,z), normalised on read (zero quaternion -> identity).
__device__ __forceinline__ Rot3 quat_to_rot(float w, float x, float y, float z)
{
    const float n2 = w * w + x * x + y * y + z * z;
    if (n2 > 0.0f) {
        const float inv = 1.0f / sqrtf(n2);
        w *= inv; x *= inv; y *= inv; z *= inv;
    } else {
        w = 1.0f; x = y = z = 0.0f;
    }
    Rot3 R;
    R.m[0] = 1.0f - 2.0f * (y * y + z * z); R.m[1] = 2.0f * (x * y - w * z);        R.m[2] = 2.0f * (x * z + w * y);
    R.m[3] = 2.0f * (x * y + w * z);        R.m[4] = 1.0f - 2.0f * (x * x + z * z); R.m[5] = 2.0f * (y * z - w * x);
    R.m[6] = 2.0f * (x * z - w * y);        R.m[7] = 2.0f * (y * z + w * x);        R.m[8] = 1.0f - 2.0f * (x * x + y * y);
    return R;
}

// A2 for the atoms of this lane: writes x into xs[c*np + i].  `sn`, `cs` hold sin/cos(theta_k).
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
        const float s = sn[k], c = cs[k];
        const float v0 = y0 - b.x, v1 = y1 - b.y, v2 = y2 - b.z;
        const float cx = u.y * v2 - u.z * v1, cy = u.z * v0 - u.x * v2, cz = u.x * v1 - u.y * v0;
        const float ud = (u.x * v0 + u.y * v1 + u.z * v2) * (1.0f - c);
        y0 = fmaf(v0, c, fmaf(cx, s, fmaf(u.x, ud, b.x)));
        y1 = fmaf(v1, c, fmaf(cy, s, fmaf(u.y, ud, b.y)));
        y2 = fmaf(v2, c, fmaf(cz, s, fmaf(u.z, ud, b.z)));
        f = __float_as_int(b.w);
    }
    x0 = fmaf(R.m[0], y0, fmaf(R.m[1], y1, fmaf(R.m[2], y2, tx)));
    x1 = fmaf(R.m[3], y0, fmaf(R.m[4], y1, fmaf(R.m[5], y2, ty)));
    x2 = fmaf(R.m[6], y0, fmaf(R.m[7], y1, fmaf(R.m[8], y2, tz)));
}

// Coordinates only (used by the top-k kernel): xs[c*np + i].
__device__ __forceinline__ void pose_coords_warp(const DevLigand &L, const float *pose, float *xs, float *sc)
{
    const int lane = threadIdx.x & 31, T = L.T, np = L.n_pad;
    float *sn = sc, *cs = sc + ((T + 3) & ~3);
    if (lane < T) {
        float s, c;
        sincosf(pose[7 + lane], &s, &c);
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

template <bool WANT_GRAD>
__device__ __noinline__ float eval_pose_warp(const DevParams &P, const DevGrid &G, const DevLigand &L,
                                             const float *pose, float *grad, float *scratch, EvalTerms *terms)
{
    const int lane = threadIdx.x & 31;
    const int N = L.N, T = L.T, np = L.n_pad;
    float *xs = scratch, *gs = scratch + 3 * np;
    float *sn = gs + 3 * np, *cs = sn + ((T + 3) & ~3);

    if (lane < T) {
        float s, c;
        sincosf(pose[7 + lane], &s, &c);
        sn[lane] = s; cs[lane] = c;
    }
    const float tx = pose[0], ty = pose[1], tz = pose[2];
    const Rot3 R = quat_to_rot(pose[3], pose[4], pose[5], pose[6]);
    __syncwarp();

    // ---- A2 + A3 -------------------------------------------------------------------------------
    float e_grid = 0.0f, e_wall = 0.0f;
    for (int i = lane; i < N; i += 32) {
        float x0, x1, x2, gx, gy, gz;
        int map_off;
        atom_coords(L, R, tx, ty, tz, sn, cs, i, x0, x1, x2, map_off);
        xs[i] = x0; xs[np + i] = x1; xs[2 * np + i] = x2;
        e_grid += atom_inter(P, G, map_off, x0, x1, x2, e_wall, gx, gy, gz);
        if (WANT_GRAD) { gs[i] = gx; gs[np + i] = gy; gs[2 * np + i] = gz; }
    }
    __syncwarp();

    // ---- A4 ------------------------------------------------------------------------------------
    float e_intra = 0.0f;
    for (int r = 0; r < L.n_rounds; ++r) {
        const float4 raw = __ldg(reinterpret_cast<const float4 *>(L.sched + r * 32 + lane));
        const int ij = __float_as_int(raw.x);
        int i = 0, j = 0;
        float fx = 0.0f, fy = 0.0f, fz = 0.0f;
        bool hit = false;
        if (ij >= 0) {
            i = ij & 0xffff; j = ij >> 16;
            const float dx = xs[i] - xs[j], dy = xs[np + i] - xs[np + j], dz = xs[2 * np + i] - xs[2 * np + j];
            const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
            if (r2 < P.cutoff2) {
                float k;
                e_intra += pair_term(P, r2, raw.y, raw.z, raw.w, k);
                fx = k * dx; fy = k * dy; fz = k * dz;
                hit = true;
            }
        }
        if (WANT_GRAD) {
            if (hit) { gs[i] += fx; gs[np + i] += fy; gs[2 * np + i] += fz; }
            __syncwarp();
            if (hit) { gs[j] -= fx; gs[np + j] -= fy; gs[2 * np + j] -= fz; }
            __syncwarp();
        }
    }

    e_grid = warp_sum(e_grid);
    e_wall = warp_sum(e_wall);
    e_intra = warp_sum(e_intra);
    if (terms) { terms->e_grid = e_grid; terms->e_wall = e_wall; terms->e_intra = e_intra; }

    // ---- A5 ------------------------------------------------------------------------------------
    if (WANT_GRAD) {
        float fx = 0.f, fy = 0.f, fz = 0.f, qx = 0.f, qy = 0.f, qz = 0.f;
        for (int i = lane; i < N; i += 32) {
            const float gx = gs[i], gy = gs[np + i], gz = gs[2 * np + i];
            const float lx = xs[i] - tx, ly = xs[np + i] - ty, lz = xs[2 * np + i] - tz;
            fx += gx; fy += gy; fz += gz;
            qx += ly * gz - lz * gy;
            qy += lz * gx - lx * gz;
            qz += lx * gy - ly * gx;
        }
        fx = warp_sum(fx); fy = warp_sum(fy); fz = warp_sum(fz);
        qx = warp_sum(qx); qy = warp_sum(qy); qz = warp_sum(qz);
        if (lane == 0) { grad[0] = fx; grad[1] = fy; grad[2] = fz; grad[3] = qx; grad[4] = qy; grad[5] = qz; }
        for (int k = 0; k < T; ++k) {
            const int2 ab = __ldg(&L.tors_ab[k]);
            const float bx = xs[ab.y], by = xs[np + ab.y], bz = xs[2 * np + ab.y];
            float ux = bx - xs[ab.x], uy = by - xs[np + ab.x], uz = bz - xs[2 * np + ab.x];
            const float inv = 1.0f / sqrtf(ux * ux + uy * uy + uz * uz);
            ux *= inv; uy *= inv; uz *= inv;
            float c = 0.0f;
            for (int i = lane; i < N; i += 32) {
                if ((__ldg(&L.atom_topo[i]).y >> k) & 1) {
                    const float gx = gs[i], gy = gs[np + i], gz = gs[2 * np + i];
                    const float lx = xs[i] - bx, ly = xs[np + i] - by, lz = xs[2 * np + i] - bz;
                    c += ux * (ly * gz - lz * gy) + uy * (lz * gx - lx * gz) + uz * (lx * gy - ly * gx);
                }
            }
            c = warp_sum(c);
            if (lane == 0) grad[6 + k] = c;
        }
        __syncwarp();
    }
    return e_grid + e_wall + e_intra;
}
