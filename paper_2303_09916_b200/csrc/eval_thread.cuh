// eval_thread.cuh -- fused pose -> coordinates -> energy + gradient, ONE THREAD PER POSE
// (eq. 2-3 at 198-219).  The throughput evaluator behind
// dock_score_batch.
//
// Why one thread per pose: all poses of a batch share the ligand, so the pair list, the torsion tree
// and every per-type constant are warp-uniform.  They live in the kernel-parameter constant bank
// (TppLigand) and are read with uniform constant loads; control flow is uniform, there are no
// shuffles, no barriers and no idle lanes, and the hydrophobic / H-bond terms are skipped by uniform
// branches for the type pairs that do not have them.  Per-thread state that needs dynamic indexing
// (coordinates, per-atom forces, sin/cos of the torsions, per-fragment force/torque) sits in shared
// memory as [row][lane] columns: conflict-free, thread-private, so no synchronisation at all.
//
//   phase 0  sin/cos of the torsions, rotation matrix, box-relative translation
//   phase 1  A2: coordinates of every atom slot (slots are the atoms sorted by fragment)
//   phase 2  A4: intra-ligand pairs, i-tiles of TPP_TILE atoms in registers; the j side is one
//            shared-memory read-modify-write per record (up to TPP_TILE pairs)
//   phase 3  A3 + A5: per atom two 16-byte gathers from the packed maps, trilinear energy and
//            gradient, wall; forces and torques accumulated per fragment about the fragment's origin
//   phase 4  A5: up-sweep over the torsion tree (children before parents): dE/dtheta_k = u_k . M_k,
//            then the fragment's force / torque are folded into its parent's
#pragma once

#include "common.cuh"
#include "mathx.cuh"

struct EvalTerms {
    float e_grid, e_wall, e_intra;
};

// floats of shared memory one WARP of the thread-per-pose evaluator needs
__host__ __device__ inline int tpp_warp_floats(int N, int T, bool want_grad)
{
    return want_grad ? 32 * (6 * N + 2 * T + 6 * (T + 1)) : 32 * (3 * N + 2 * T);
}

template <bool SCHED_PARAM>
__device__ __forceinline__ uint32_t tpp_word(const TppLigand &L, int pos)
{
    return SCHED_PARAM ? L.sched[pos] : __ldg(L.sched_global + pos);
}

// pose[k * ps] = k-th pose component of this thread; grad[k * gs] receives the k-th gradient component.
// `sm` = this warp's shared memory (tpp_warp_floats floats).  Returns E = e_grid + e_wall + e_intra.
template <bool WANT_GRAD, bool SCHED_PARAM>
__device__ __forceinline__ float eval_pose_thread(const DevParams &P, const DevGrid &G, const TppLigand &L,
                                                  const float *__restrict__ pose, int ps,
                                                  float *__restrict__ grad, int gs,
                                                  float *__restrict__ sm, EvalTerms &terms)
{
    const int lane = threadIdx.x & 31;
    const int N = L.N, T = L.T;
    float2 *const xy = reinterpret_cast<float2 *>(sm) + lane;                  // [N]   stride 32
    float *const zz = sm + 64 * N + lane;                                      // [N]
    float2 *const sc = reinterpret_cast<float2 *>(sm + 96 * N) + lane;         // [T]   {sin, cos}
    float2 *const gxy = reinterpret_cast<float2 *>(sm + 96 * N + 64 * T) + lane;   // [N]
    float *const gz = sm + 160 * N + 64 * T + lane;                            // [N]
    float2 *const fm = reinterpret_cast<float2 *>(sm + 192 * N + 64 * T) + lane;   // [T+1][3]: (Fx,Fy) (Fz,Mx) (My,Mz)

    // ---- phase 0 ---------------------------------------------------------------------------------
    for (int k = 0; k < T; ++k) {
        float s, c;
        sincos_cw(pose[(7 + k) * ps], s, c);
        sc[k * 32] = make_float2(s, c);
    }
    const float tx = (pose[0] - G.rx) - G.rdx;
    const float ty = (pose[ps] - G.ry) - G.rdy;
    const float tz = (pose[2 * ps] - G.rz) - G.rdz;
    const Rot3 R = quat_to_rot(pose[3 * ps], pose[4 * ps], pose[5 * ps], pose[6 * ps]);

    // ---- phase 1: A2 -------------------------------------------------------------------------------
    for (int s = 0; s < N; ++s) {
        const float4 a = L.atom_ref[s];
        float y0 = a.x, y1 = a.y, y2 = a.z;
        int f = L.atom_frag[s];
        while (f > 0) {
            const float4 u = L.tors_axis[f - 1];
            const float4 b = L.tors_pt[f - 1];
            const float2 v = sc[(f - 1) * 32];
            rodrigues(u.x, u.y, u.z, b.x, b.y, b.z, v.x, v.y, 1.0f - v.y, y0, y1, y2);
            f = __float_as_int(u.w);
        }
        const float x0 = fmaf(R.m00, y0, fmaf(R.m01, y1, fmaf(R.m02, y2, tx)));
        const float x1 = fmaf(R.m10, y0, fmaf(R.m11, y1, fmaf(R.m12, y2, ty)));
        const float x2 = fmaf(R.m20, y0, fmaf(R.m21, y1, fmaf(R.m22, y2, tz)));
        xy[s * 32] = make_float2(x0, x1);
        zz[s * 32] = x2;
        if (WANT_GRAD) {
            gxy[s * 32] = make_float2(0.0f, 0.0f);
            gz[s * 32] = 0.0f;
        }
    }

    // ---- phase 2: A4 -------------------------------------------------------------------------------
    float e_intra = 0.0f;
    {
        int pos = 0;
        for (int g = 0; g < L.n_groups; ++g) {
            const uint32_t h0 = tpp_word<SCHED_PARAM>(L, pos), h1 = tpp_word<SCHED_PARAM>(L, pos + 1);
            pos += 2;
            const int n_rec = (int)(h1 & 0xffffu), n_i = (int)(h1 >> 16);
            float xi[TPP_TILE], yi[TPP_TILE], zi[TPP_TILE], fxi[TPP_TILE], fyi[TPP_TILE], fzi[TPP_TILE];
#pragma unroll
            for (int t = 0; t < TPP_TILE; ++t) {
                const int i = (int)((h0 >> (8 * t)) & 0xffu);
                const float2 a = xy[i * 32];
                xi[t] = a.x; yi[t] = a.y; zi[t] = zz[i * 32];
                fxi[t] = fyi[t] = fzi[t] = 0.0f;
            }
            for (int r = 0; r < n_rec; ++r) {
                const uint32_t w0 = tpp_word<SCHED_PARAM>(L, pos);
                const int j = (int)(w0 & 0xffu);
                const float2 b = xy[j * 32];
                const float bz = zz[j * 32];
                float fxj = 0.0f, fyj = 0.0f, fzj = 0.0f;
#pragma unroll
                for (int t = 0; t < TPP_TILE; ++t) {
                    if (w0 & (0x100u << t)) {                                   // uniform: pair (i_t, j) is listed
                        const float rsum = __uint_as_float(tpp_word<SCHED_PARAM>(L, pos + 1 + t));
                        const float dx = xi[t] - b.x, dy = yi[t] - b.y, dz = zi[t] - bz;
                        const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
                        float k, e;
                        const bool hyd = (w0 & (0x1000u << t)) != 0, hb = (w0 & (0x10000u << t)) != 0;   // uniform
                        if (!hyd && !hb) e = pair_term<false, false>(P, r2, rsum, k);
                        else if (hyd && !hb) e = pair_term<true, false>(P, r2, rsum, k);
                        else if (!hyd) e = pair_term<false, true>(P, r2, rsum, k);
                        else e = pair_term<true, true>(P, r2, rsum, k);
                        if (r2 < P.cutoff2) {
                            e_intra += e;
                            if (WANT_GRAD) {
                                const float fx = k * dx, fy = k * dy, fz = k * dz;
                                fxi[t] += fx; fyi[t] += fy; fzi[t] += fz;
                                fxj -= fx; fyj -= fy; fzj -= fz;
                            }
                        }
                    }
                }
                if (WANT_GRAD) {
                    float2 gj = gxy[j * 32];
                    gj.x += fxj; gj.y += fyj;
                    gxy[j * 32] = gj;
                    gz[j * 32] += fzj;
                }
                pos += TPP_REC_WORDS;
            }
            if (WANT_GRAD) {
#pragma unroll
                for (int t = 0; t < TPP_TILE; ++t) {
                    if (t < n_i) {
                        const int i = (int)((h0 >> (8 * t)) & 0xffu);
                        float2 gi = gxy[i * 32];
                        gi.x += fxi[t]; gi.y += fyi[t];
                        gxy[i * 32] = gi;
                        gz[i * 32] += fzi[t];
                    }
                }
            }
        }
    }

    // ---- phase 3: A3 (+ per-fragment force / torque sums of A5) ----------------------------------------
    float e_grid = 0.0f, e_wall = 0.0f;
    {
        constexpr int CH = 4;                   // atoms whose gathers are in flight together
        int f = 0, f_end = L.frag_end[0];
        float ox = tx, oy = ty, oz = tz;        // origin of the current fragment (root: the pivot)
        float Fx = 0.f, Fy = 0.f, Fz = 0.f, Mx = 0.f, My = 0.f, Mz = 0.f;
        for (int s0 = 0; s0 < N; s0 += CH) {
            CellRef cr[CH];
            float4 q0[CH], q1[CH];
            float px[CH], py[CH], pz[CH];
#pragma unroll
            for (int a = 0; a < CH; ++a) {
                const int s = min(s0 + a, N - 1);
                const float2 v = xy[s * 32];
                px[a] = v.x; py[a] = v.y; pz[a] = zz[s * 32];
                cr[a] = locate_cell(G, px[a], py[a], pz[a]);
                const float4 *e0 = G.packed + (size_t)__float_as_int(L.atom_ref[s].w) + cr[a].idx;
                q0[a] = __ldg(e0);
                q1[a] = __ldg(e0 + G.nx * G.ny);
            }
#pragma unroll
            for (int a = 0; a < CH; ++a) {
                const int s = s0 + a;
                if (s < N) {
                    float gx, gy, gz_;
                    e_grid += trilinear(G, cr[a], q0[a], q1[a], e_wall, gx, gy, gz_);
                    if (WANT_GRAD) {
                        while (s == f_end) {                                   // uniform: next fragment starts at slot s
                            fm[(3 * f) * 32] = make_float2(Fx, Fy);
                            fm[(3 * f + 1) * 32] = make_float2(Fz, Mx);
                            fm[(3 * f + 2) * 32] = make_float2(My, Mz);
                            ++f;
                            f_end = L.frag_end[f];
                            const int bs = L.tors_b[f - 1];
                            const float2 ob = xy[bs * 32];
                            ox = ob.x; oy = ob.y; oz = zz[bs * 32];
                            Fx = Fy = Fz = Mx = My = Mz = 0.f;
                        }
                        const float2 gp = gxy[s * 32];
                        gx += gp.x; gy += gp.y; gz_ += gz[s * 32];
                        const float lx = px[a] - ox, ly = py[a] - oy, lz = pz[a] - oz;
                        Fx += gx; Fy += gy; Fz += gz_;
                        Mx = fmaf(ly, gz_, fmaf(-lz, gy, Mx));
                        My = fmaf(lz, gx, fmaf(-lx, gz_, My));
                        Mz = fmaf(lx, gy, fmaf(-ly, gx, Mz));
                    }
                }
            }
        }
        if (WANT_GRAD) {
            fm[(3 * f) * 32] = make_float2(Fx, Fy);
            fm[(3 * f + 1) * 32] = make_float2(Fz, Mx);
            fm[(3 * f + 2) * 32] = make_float2(My, Mz);
        }
    }

    // ---- phase 4: A5 up-sweep --------------------------------------------------------------------------
    if (WANT_GRAD) {
        for (int f = T; f >= 1; --f) {
            const float2 a0 = fm[(3 * f) * 32], a1 = fm[(3 * f + 1) * 32], a2 = fm[(3 * f + 2) * 32];
            const float Fx = a0.x, Fy = a0.y, Fz = a1.x, Mx = a1.y, My = a2.x, Mz = a2.y;
            const int as = L.tors_a[f - 1], bs = L.tors_b[f - 1];
            const float4 tp = L.tors_pt[f - 1];
            const float2 xb = xy[bs * 32], xa = xy[as * 32];
            const float zb = zz[bs * 32], za = zz[as * 32];
            const float ux = (xb.x - xa.x) * tp.w, uy = (xb.y - xa.y) * tp.w, uz = (zb - za) * tp.w;   // lab-frame unit axis
            grad[(6 + f - 1) * gs] = fmaf(ux, Mx, fmaf(uy, My, uz * Mz));
            const int p = __float_as_int(L.tors_axis[f - 1].w);                 // parent fragment
            float pox = tx, poy = ty, poz = tz;
            if (p > 0) {
                const int pb = L.tors_b[p - 1];
                const float2 o = xy[pb * 32];
                pox = o.x; poy = o.y; poz = zz[pb * 32];
            }
            const float lx = xb.x - pox, ly = xb.y - poy, lz = zb - poz;
            float2 b0 = fm[(3 * p) * 32], b1 = fm[(3 * p + 1) * 32], b2 = fm[(3 * p + 2) * 32];
            b0.x += Fx; b0.y += Fy; b1.x += Fz;
            b1.y += Mx + fmaf(ly, Fz, -lz * Fy);
            b2.x += My + fmaf(lz, Fx, -lx * Fz);
            b2.y += Mz + fmaf(lx, Fy, -ly * Fx);
            fm[(3 * p) * 32] = b0; fm[(3 * p + 1) * 32] = b1; fm[(3 * p + 2) * 32] = b2;
        }
        const float2 a0 = fm[0], a1 = fm[32], a2 = fm[64];
        grad[0] = a0.x; grad[gs] = a0.y; grad[2 * gs] = a1.x;
        grad[3 * gs] = a1.y; grad[4 * gs] = a2.x; grad[5 * gs] = a2.y;
    }
    terms.e_grid = e_grid; terms.e_wall = e_wall; terms.e_intra = e_intra;
    return e_grid + e_wall + e_intra;
}
