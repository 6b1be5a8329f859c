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
// Shared memory bounds the occupancy (about 7 warps per SM for a 30-atom ligand), so the kernel is
// written for instruction-level parallelism instead: the pair phase is branch-free straight-line
// code over 8 independent pairs (2 partner atoms x a 4-atom register tile) that the scheduler can
// interleave (profiles/r1a.md -> r1c.md).
//
//   phase 1  A2: one rigid frame (rotation + offset) per fragment, parents first, composed from the
//            parent's frame and one Rodrigues rotation; atoms of a fragment are 9 FMAs each.
//            Coordinates are stored RELATIVE TO THE PIVOT (smaller numbers -> smaller fp32 error in
//            pair distances and lever arms); the translation is added for the grid lookup only.
//   phase 2  A4: intra-ligand pairs (schedule format: common.cuh); the weights of the two Gaussians
//            are folded into the exponent arguments, unlisted pairs are masked through their data.
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

// floats of shared memory one THREAD of the evaluator needs:
//   [xy: 2N][z: N][R: max(3N, 12(T+1))  per-atom forces, aliased by the fragment frames in phase 1][fm: 6(T+1)]
__host__ __device__ inline int tpp_thread_floats(int N, int T, bool want_grad)
{
    const int frames = 12 * (T + 1);
    if (!want_grad) return 3 * N + frames;
    return 3 * N + (3 * N > frames ? 3 * N : frames) + 6 * (T + 1);
}
__host__ __device__ inline int tpp_warp_floats(int N, int T, bool want_grad)
{
    return 32 * tpp_thread_floats(N, T, want_grad);
}

template <bool SCHED_PARAM>
__device__ __forceinline__ uint4 tpp_quad(const TppLigand &L, int pos)
{
    return SCHED_PARAM ? L.sched[pos] : __ldg(L.sched_global + pos);
}

// Energy accumulators of the pair phase; E_intra = s1 g1 + s2 g2 + rep/2 + lin.
struct PairAcc {
    float g1, g2, rep, lin;
};

// One pair (i, j): d = r - rsum; accumulates the energy terms and the force k (x_i - x_j) on i, -that on j.
// rsum = TPP_MASKED_RSUM makes every term exactly 0.  SPECIAL adds the hydrophobic and H-bond ramps with the
// per-pair weights wh, whb (0 where the type pair has none).
template <bool SPECIAL, bool WANT_GRAD>
__device__ __forceinline__ void pair_eval(const DevParams &P, float xi, float yi, float zi, float xj, float yj, float zj,
                                          float rsum, float wh, float whb, PairAcc &acc,
                                          float &fxi, float &fyi, float &fzi, float &fxj, float &fyj, float &fzj)
{
    const float dx = xi - xj, dy = yi - yj, dz = zi - zj;
    const float r2 = fmaf(dz, dz, fmaf(dy, dy, fmaf(dx, dx, 1e-12f)));
    const float rinv = fast_rsqrt(r2);
    // out of range (r >= cutoff, decided on r^2 in fp32) -> the same "infinitely far" surface distance as a masked
    // pair: every term and derivative below is then exactly 0, with no branch in the instruction stream
    const float d = (r2 < P.cutoff2) ? fmaf(r2, rinv, -rsum) : 1.0e18f;
    const float g1 = fast_ex2(fmaf(d * -5.770780163555854f, d, P.lw1));        // |w1| exp(-(d/0.5)^2)
    const float b = d - 3.0f;
    const float g2 = fast_ex2(fmaf(b * -0.36067376022224085f, b, P.lw2));      // |w2| exp(-((d-3)/2)^2)
    const float m = fminf(d, 0.0f);
    const float m2 = m * P.w3x2;                                                // 2 w3 min(d,0)
    float de = fmaf(P.k1, d * g1, fmaf(P.k2, b * g2, m2));                      // dE/dd
    acc.g1 += g1;
    acc.g2 += g2;
    acc.rep = fmaf(m2, m, acc.rep);
    if (SPECIAL) {
        const float th = 1.5f - d, hh = __saturatef(th);                        // hydrophobic: 1 | 1.5 - d | 0
        const float tb = d * -1.4285714285714286f, hb = __saturatef(tb);        // H-bond:      1 | -d/0.7  | 0
        acc.lin = fmaf(wh, hh, fmaf(whb, hb, acc.lin));
        de -= (hh == th) ? wh : 0.0f;                                           // on the ramp iff the clamp did nothing
        de = fmaf((hb == tb) ? whb : 0.0f, -1.4285714285714286f, de);
    }
    if (WANT_GRAD) {
        const float k = de * rinv;
        fxi = fmaf(k, dx, fxi); fyi = fmaf(k, dy, fyi); fzi = fmaf(k, dz, fzi);
        fxj = fmaf(-k, dx, fxj); fyj = fmaf(-k, dy, fyj); fzj = fmaf(-k, dz, fzj);
    }
}

// The register tile of the pair phase: TPP_TILE atoms with their force accumulators.
struct PairTile {
    float x[TPP_TILE], y[TPP_TILE], z[TPP_TILE], fx[TPP_TILE], fy[TPP_TILE], fz[TPP_TILE];
};

// One record: partner column at byte offset `off` (z column; the (x,y) column is at 2*off) against the tile.
template <bool SPECIAL, bool WANT_GRAD, bool SCHED_PARAM>
__device__ __forceinline__ void record_single(const DevParams &P, const TppLigand &L, int &pos, PairTile &t, PairAcc &acc,
                                              const char *xy, const char *zz, char *gxy, char *gz)
{
    const uint4 h = tpp_quad<SCHED_PARAM>(L, pos);
    const uint4 qr = tpp_quad<SCHED_PARAM>(L, pos + 1);
    uint4 qh = make_uint4(0, 0, 0, 0), qb = make_uint4(0, 0, 0, 0);
    if (SPECIAL) { qh = tpp_quad<SCHED_PARAM>(L, pos + 2); qb = tpp_quad<SCHED_PARAM>(L, pos + 3); }
    pos += SPECIAL ? 4 : 2;
    const float2 bj = *reinterpret_cast<const float2 *>(xy + 2 * h.x);
    const float bz = *reinterpret_cast<const float *>(zz + h.x);
    float2 gj = make_float2(0.f, 0.f);
    float gjz = 0.f;
    if (WANT_GRAD) { gj = *reinterpret_cast<float2 *>(gxy + 2 * h.x); gjz = *reinterpret_cast<float *>(gz + h.x); }
    const float rs[4] = {__uint_as_float(qr.x), __uint_as_float(qr.y), __uint_as_float(qr.z), __uint_as_float(qr.w)};
    const float wh[4] = {__uint_as_float(qh.x), __uint_as_float(qh.y), __uint_as_float(qh.z), __uint_as_float(qh.w)};
    const float wb[4] = {__uint_as_float(qb.x), __uint_as_float(qb.y), __uint_as_float(qb.z), __uint_as_float(qb.w)};
#pragma unroll
    for (int k = 0; k < TPP_TILE; ++k)
        pair_eval<SPECIAL, WANT_GRAD>(P, t.x[k], t.y[k], t.z[k], bj.x, bj.y, bz, rs[k], wh[k], wb[k], acc,
                                      t.fx[k], t.fy[k], t.fz[k], gj.x, gj.y, gjz);
    if (WANT_GRAD) {
        *reinterpret_cast<float2 *>(gxy + 2 * h.x) = gj;
        *reinterpret_cast<float *>(gz + h.x) = gjz;
    }
}

// Two records at once: 8 independent pairs in flight (the partner columns are distinct slots).
template <bool SPECIAL, bool WANT_GRAD, bool SCHED_PARAM>
__device__ __forceinline__ void record_double(const DevParams &P, const TppLigand &L, int &pos, PairTile &t,
                                              PairAcc &accA, PairAcc &accB,
                                              const char *xy, const char *zz, char *gxy, char *gz)
{
    constexpr int S = SPECIAL ? 3 : 1;
    const uint4 h = tpp_quad<SCHED_PARAM>(L, pos);
    const uint4 qrA = tpp_quad<SCHED_PARAM>(L, pos + 1), qrB = tpp_quad<SCHED_PARAM>(L, pos + 1 + S);
    uint4 qhA = make_uint4(0, 0, 0, 0), qbA = qhA, qhB = qhA, qbB = qhA;
    if (SPECIAL) {
        qhA = tpp_quad<SCHED_PARAM>(L, pos + 2); qbA = tpp_quad<SCHED_PARAM>(L, pos + 3);
        qhB = tpp_quad<SCHED_PARAM>(L, pos + 5); qbB = tpp_quad<SCHED_PARAM>(L, pos + 6);
    }
    pos += 1 + 2 * S;
    const float2 a = *reinterpret_cast<const float2 *>(xy + 2 * h.x);
    const float az = *reinterpret_cast<const float *>(zz + h.x);
    const float2 b = *reinterpret_cast<const float2 *>(xy + 2 * h.y);
    const float bz = *reinterpret_cast<const float *>(zz + h.y);
    float2 ga = make_float2(0.f, 0.f), gb = ga;
    float gaz = 0.f, gbz = 0.f;
    if (WANT_GRAD) {
        ga = *reinterpret_cast<float2 *>(gxy + 2 * h.x); gaz = *reinterpret_cast<float *>(gz + h.x);
        gb = *reinterpret_cast<float2 *>(gxy + 2 * h.y); gbz = *reinterpret_cast<float *>(gz + h.y);
    }
    const float rA[4] = {__uint_as_float(qrA.x), __uint_as_float(qrA.y), __uint_as_float(qrA.z), __uint_as_float(qrA.w)};
    const float rB[4] = {__uint_as_float(qrB.x), __uint_as_float(qrB.y), __uint_as_float(qrB.z), __uint_as_float(qrB.w)};
    const float hA[4] = {__uint_as_float(qhA.x), __uint_as_float(qhA.y), __uint_as_float(qhA.z), __uint_as_float(qhA.w)};
    const float hB[4] = {__uint_as_float(qhB.x), __uint_as_float(qhB.y), __uint_as_float(qhB.z), __uint_as_float(qhB.w)};
    const float bA[4] = {__uint_as_float(qbA.x), __uint_as_float(qbA.y), __uint_as_float(qbA.z), __uint_as_float(qbA.w)};
    const float bB[4] = {__uint_as_float(qbB.x), __uint_as_float(qbB.y), __uint_as_float(qbB.z), __uint_as_float(qbB.w)};
#pragma unroll
    for (int k = 0; k < TPP_TILE; ++k) {
        pair_eval<SPECIAL, WANT_GRAD>(P, t.x[k], t.y[k], t.z[k], a.x, a.y, az, rA[k], hA[k], bA[k], accA,
                                      t.fx[k], t.fy[k], t.fz[k], ga.x, ga.y, gaz);
        pair_eval<SPECIAL, WANT_GRAD>(P, t.x[k], t.y[k], t.z[k], b.x, b.y, bz, rB[k], hB[k], bB[k], accB,
                                      t.fx[k], t.fy[k], t.fz[k], gb.x, gb.y, gbz);
    }
    if (WANT_GRAD) {
        *reinterpret_cast<float2 *>(gxy + 2 * h.x) = ga;
        *reinterpret_cast<float *>(gz + h.x) = gaz;
        *reinterpret_cast<float2 *>(gxy + 2 * h.y) = gb;
        *reinterpret_cast<float *>(gz + h.y) = gbz;
    }
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
    const int rg = WANT_GRAD ? max(3 * N, 12 * (T + 1)) : 12 * (T + 1);
    float2 *const xy = reinterpret_cast<float2 *>(sm) + lane;                      // [N]   stride 32
    float *const zz = sm + 64 * N + lane;                                          // [N]
    float *const rbase = sm + 96 * N;
    float2 *const fr = reinterpret_cast<float2 *>(rbase) + lane;                   // [T+1][6] frames (phase 1 only)
    float2 *const gxy = reinterpret_cast<float2 *>(rbase) + lane;                  // [N]
    float *const gz = rbase + 64 * N + lane;                                       // [N]
    float2 *const fm = reinterpret_cast<float2 *>(rbase + 32 * rg) + lane;         // [T+1][3]: (Fx,Fy) (Fz,Mx) (My,Mz)

    const float tx = (pose[0] - G.rx) - G.rdx;
    const float ty = (pose[ps] - G.ry) - G.rdy;
    const float tz = (pose[2 * ps] - G.rz) - G.rdz;

    // ---- phase 1: A2 -------------------------------------------------------------------------------
    {
        Rot3 A = quat_to_rot(pose[3 * ps], pose[4 * ps], pose[5 * ps], pose[6 * ps]);
        float c0 = 0.0f, c1 = 0.0f, c2 = 0.0f;                                     // pivot-relative
        int s = 0;
        for (int f = 0; f <= T; ++f) {
            if (f > 0) {
                const int k = f - 1;
                const float4 u = L.tors_axis[k];
                const float4 b = L.tors_pt[k];
                const int p = __float_as_int(u.w);
                const float2 p0 = fr[(6 * p) * 32], p1 = fr[(6 * p + 1) * 32], p2 = fr[(6 * p + 2) * 32];
                const float2 p3 = fr[(6 * p + 3) * 32], p4 = fr[(6 * p + 4) * 32], p5 = fr[(6 * p + 5) * 32];
                float sn, cs;
                sincos_cw(pose[(7 + k) * ps], sn, cs);
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

    // ---- phase 2: A4 -------------------------------------------------------------------------------
    float e_intra = 0.0f;
    {
        const char *xyb = reinterpret_cast<const char *>(xy), *zzb = reinterpret_cast<const char *>(zz);
        char *gxyb = reinterpret_cast<char *>(gxy), *gzb = reinterpret_cast<char *>(gz);
        PairAcc accA = {0.f, 0.f, 0.f, 0.f}, accB = {0.f, 0.f, 0.f, 0.f};
        int pos = 0;
        for (int g = 0; g < L.n_groups; ++g) {
            const uint4 hdr = tpp_quad<SCHED_PARAM>(L, pos++);
            PairTile t;
#pragma unroll
            for (int k = 0; k < TPP_TILE; ++k) {
                const int i = (int)((hdr.x >> (8 * k)) & 0xffu);
                const float2 a = xy[i * 32];
                t.x[k] = a.x; t.y[k] = a.y; t.z[k] = zz[i * 32];
                t.fx[k] = t.fy[k] = t.fz[k] = 0.0f;
            }
            const int np2 = (int)(hdr.y & 0xffffu), np1 = (int)(hdr.y >> 16);
            const int ns2 = (int)(hdr.z & 0xffffu), ns1 = (int)(hdr.z >> 16);
            for (int r = 0; r < np2; ++r) record_double<false, WANT_GRAD, SCHED_PARAM>(P, L, pos, t, accA, accB, xyb, zzb, gxyb, gzb);
            if (np1) record_single<false, WANT_GRAD, SCHED_PARAM>(P, L, pos, t, accA, xyb, zzb, gxyb, gzb);
            for (int r = 0; r < ns2; ++r) record_double<true, WANT_GRAD, SCHED_PARAM>(P, L, pos, t, accA, accB, xyb, zzb, gxyb, gzb);
            if (ns1) record_single<true, WANT_GRAD, SCHED_PARAM>(P, L, pos, t, accA, xyb, zzb, gxyb, gzb);
            if (WANT_GRAD) {
                // padding slots of the last tile repeat its first slot with all pairs masked: they add exact zeros
#pragma unroll
                for (int k = 0; k < TPP_TILE; ++k) {
                    const int i = (int)((hdr.x >> (8 * k)) & 0xffu);
                    float2 gi = gxy[i * 32];
                    gi.x += t.fx[k]; gi.y += t.fy[k];
                    gxy[i * 32] = gi;
                    gz[i * 32] += t.fz[k];
                }
            }
        }
        e_intra = fmaf(P.s1, accA.g1 + accB.g1, fmaf(P.s2, accA.g2 + accB.g2, fmaf(0.5f, accA.rep + accB.rep, accA.lin + accB.lin)));
    }

    // ---- phase 3: A3 (+ per-fragment force / torque sums of A5) ----------------------------------------
    float e_grid = 0.0f, e_wall = 0.0f;
    {
        constexpr int CH = 4;                   // atoms whose gathers are in flight together
        int f = 0, f_end = L.frag_end[0];
        float ox = 0.0f, oy = 0.0f, oz = 0.0f;  // origin of the current fragment (root: the pivot), pivot-relative
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
                cr[a] = locate_cell(G, px[a] + tx, py[a] + ty, pz[a] + tz);
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
            // fragments after the last atom-bearing one cannot exist (every fragment owns atom b), so f == T here
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
            float pox = 0.0f, poy = 0.0f, poz = 0.0f;
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
