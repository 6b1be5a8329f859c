// mathx.cuh -- scalar building blocks shared by the two evaluators (thread-per-pose and
// warp-per-pose): sine/cosine without a slow path, quaternion -> rotation, the Vina-style pair term
// and the trilinear interpolant with its partial derivatives (eq. 2-3,
// 198-219) on the packed gather layout.  Product code; shares nothing with oracle/.
#pragma once

#include "common.cuh"

// sin and cos of x for |x| < 1.2e4 rad, ~1 ulp: Cody-Waite reduction to [-pi/4, pi/4] with pi/2 split
// into 11-bit chunks (k * chunk is exact for |k| < 2^13), then the classic single-precision minimax
// polynomials.  No table, no local memory, no divergent slow path.
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
    ps = fmaf(ps * z, r, r);                                   // sin(r)
    float pc = fmaf(z, 2.443315711809948e-5f, -1.388731625493765e-3f);
    pc = fmaf(pc, z, 4.166664568298827e-2f);
    pc = fmaf(pc * z, z, fmaf(-0.5f, z, 1.0f));                // cos(r)
    const float ss = (q & 1) ? pc : ps;
    const float cc = (q & 1) ? ps : pc;
    s = (q & 2) ? -ss : ss;
    c = ((q + 1) & 2) ? -cc : cc;
}

struct Rot3 {
    float m00, m01, m02, m10, m11, m12, m20, m21, m22;
};

// q = (w,x,y,z), normalised on read (zero quaternion -> identity).
__device__ __forceinline__ Rot3 quat_to_rot(float w, float x, float y, float z)
{
    const float n2 = fmaf(w, w, fmaf(x, x, fmaf(y, y, z * z)));
    if (n2 > 0.0f) {
        const float inv = 1.0f / sqrtf(n2);
        w *= inv; x *= inv; y *= inv; z *= inv;
    } else {
        w = 1.0f; x = y = z = 0.0f;
    }
    Rot3 R;
    const float x2 = x + x, y2 = y + y, z2 = z + z;
    R.m00 = 1.0f - fmaf(y2, y, z2 * z); R.m01 = fmaf(x2, y, -w * z2);       R.m02 = fmaf(x2, z, w * y2);
    R.m10 = fmaf(x2, y, w * z2);        R.m11 = 1.0f - fmaf(x2, x, z2 * z); R.m12 = fmaf(y2, z, -w * x2);
    R.m20 = fmaf(x2, z, -w * y2);       R.m21 = fmaf(y2, z, w * x2);        R.m22 = 1.0f - fmaf(x2, x, y2 * y);
    return R;
}

// One Rodrigues rotation of y about the axis (ux,uy,uz) through (bx,by,bz) by the angle with
// sine s and cosine c (omc = 1 - c):  y <- b + v c + (u x v) s + u (u.v)(1-c),  v = y - b.
__device__ __forceinline__ void rodrigues(float ux, float uy, float uz, float bx, float by, float bz,
                                          float s, float c, float omc, float &y0, float &y1, float &y2)
{
    const float v0 = y0 - bx, v1 = y1 - by, v2 = y2 - bz;
    const float cx = fmaf(uy, v2, -uz * v1), cy = fmaf(uz, v0, -ux * v2), cz = fmaf(ux, v1, -uy * v0);
    const float ud = fmaf(ux, v0, fmaf(uy, v1, uz * v2)) * omc;
    y0 = fmaf(v0, c, fmaf(cx, s, fmaf(ux, ud, bx)));
    y1 = fmaf(v1, c, fmaf(cy, s, fmaf(uy, ud, by)));
    y2 = fmaf(v2, c, fmaf(cz, s, fmaf(uz, ud, bz)));
}

// Vina-style pair term on the surface distance d = r - (R_i + R_j), for r2 < cutoff^2
// (the caller decides the cutoff).  HYD / HB say whether the hydrophobic / H-bond terms apply to
// this type pair.  Returns e; k = (de/dr)/r so that the force on atom i is k * (x_i - x_j).
template <bool HYD, bool HB>
__device__ __forceinline__ float pair_term(const DevParams &P, float r2, float rsum, float &k)
{
    r2 = fmaxf(r2, 1e-12f);
    const float rinv = fast_rsqrt(r2);
    const float d = fmaf(r2, rinv, -rsum);
    const float g1 = fast_ex2(d * d * -5.770780163555854f);              // exp(-(d/0.5)^2)
    const float b = d - 3.0f;
    const float g2 = fast_ex2(b * b * -0.36067376022224085f);            // exp(-((d-3)/2)^2)
    const float m = fminf(d, 0.0f);
    const float w1g1 = P.w[0] * g1, w2g2 = P.w[1] * g2, w3m = P.w[2] * m;
    float e = fmaf(w3m, m, w1g1 + w2g2);
    float de = fmaf(-8.0f * d, w1g1, fmaf(-0.5f * b, w2g2, w3m + w3m));
    if (HYD) {                                                          // 1 | 1.5 - d | 0
        e = fmaf(P.w[3], __saturatef(1.5f - d), e);
        de -= (d >= 0.5f && d < 1.5f) ? P.w[3] : 0.0f;
    }
    if (HB) {                                                           // 1 | -d/0.7 | 0
        e = fmaf(P.w[4], __saturatef(d * -1.4285714285714286f), e);
        de -= (d >= -0.7f && d < 0.0f) ? P.w[4] * 1.4285714285714286f : 0.0f;
    }
    k = de * rinv;
    return e;
}

// Runtime-flag variant for the warp-per-pose evaluator, where every lane holds a different pair:
// wh = w4 or 0, whb = w5 or 0.
__device__ __forceinline__ float pair_term_rt(const DevParams &P, float r2, float rsum, float wh, float whb, float &k)
{
    r2 = fmaxf(r2, 1e-12f);
    const float rinv = fast_rsqrt(r2);
    const float d = fmaf(r2, rinv, -rsum);
    const float g1 = fast_ex2(d * d * -5.770780163555854f);
    const float b = d - 3.0f;
    const float g2 = fast_ex2(b * b * -0.36067376022224085f);
    const float m = fminf(d, 0.0f);
    const float w1g1 = P.w[0] * g1, w2g2 = P.w[1] * g2, w3m = P.w[2] * m;
    float e = fmaf(w3m, m, w1g1 + w2g2);
    e = fmaf(wh, __saturatef(1.5f - d), e);
    e = fmaf(whb, __saturatef(d * -1.4285714285714286f), e);
    float de = fmaf(-8.0f * d, w1g1, fmaf(-0.5f * b, w2g2, w3m + w3m));
    de -= (d >= 0.5f && d < 1.5f) ? wh : 0.0f;
    de -= (d >= -0.7f && d < 0.0f) ? whb * 1.4285714285714286f : 0.0f;
    k = de * rinv;
    return e;
}

// Cell lookup of one atom at the box-relative position (x,y,z) [A, relative to the lattice's
// reference node, see DevGrid].  Produces the flat entry index, the in-cell fractions p (eq. 2's
// p_x,p_y,p_z) and the overshoot outside the box in cell units (0 inside).
struct CellRef {
    int   idx;            // entry index into one map of DevGrid::packed
    float px, py, pz;
    float ox, oy, oz;     // overshoot in cells (signed); 0 inside the box
};

__device__ __forceinline__ CellRef locate_cell(const DevGrid &G, float x, float y, float z)
{
    // u = x / h with the rounding error of inv_h removed by its low word
    const float ux = fmaf(x, G.inv_h_lo, x * G.inv_h);
    const float uy = fmaf(y, G.inv_h_lo, y * G.inv_h);
    const float uz = fmaf(z, G.inv_h_lo, z * G.inv_h);
    const float cx = fminf(fmaxf(ux, G.lo_x), G.hi_x);
    const float cy = fminf(fmaxf(uy, G.lo_y), G.hi_y);
    const float cz = fminf(fmaxf(uz, G.lo_z), G.hi_z);
    CellRef c;
    c.ox = ux - cx; c.oy = uy - cy; c.oz = uz - cz;
    const float fx = fminf(floorf(cx), G.hi_x - 1.0f);      // i0 = min(floor(u), n-2): reading S8
    const float fy = fminf(floorf(cy), G.hi_y - 1.0f);
    const float fz = fminf(floorf(cz), G.hi_z - 1.0f);
    c.px = cx - fx; c.py = cy - fy; c.pz = cz - fz;
    const int ix = (int)fx + G.icx, iy = (int)fy + G.icy, iz = (int)fz + G.icz;
    c.idx = (iz * G.ny + iy) * G.nx + ix;
    return c;
}

// Clamped axes get zero grid gradient and the quadratic wall (reading S7).  ggx.. in kcal/mol/A.
__device__ __forceinline__ void apply_wall(const DevGrid &G, const CellRef &c, float ggx, float ggy, float ggz,
                                           float &e_wall, float &gx, float &gy, float &gz)
{
    if (c.ox != 0.0f) ggx = 0.0f;
    if (c.oy != 0.0f) ggy = 0.0f;
    if (c.oz != 0.0f) ggz = 0.0f;
    gx = fmaf(G.kw_g, c.ox, ggx);                                                     // 2 k h * overshoot_cells
    gy = fmaf(G.kw_g, c.oy, ggy);
    gz = fmaf(G.kw_g, c.oz, ggz);
    e_wall = fmaf(G.kw_e, fmaf(c.ox, c.ox, fmaf(c.oy, c.oy, c.oz * c.oz)), e_wall);   // k h^2 * sum overshoot_cells^2
}

// Value of the trilinear interpolant (eq. 2) of one channel from its packed cell.
__device__ __forceinline__ float trilerp(const CellRef &c, const float4 q0, const float4 q1)
{
    const float c00 = fmaf(c.px, q0.y - q0.x, q0.x), c10 = fmaf(c.px, q0.w - q0.z, q0.z);
    const float c01 = fmaf(c.px, q1.y - q1.x, q1.x), c11 = fmaf(c.px, q1.w - q1.z, q1.z);
    const float c0 = fmaf(c.py, c10 - c00, c00), c1 = fmaf(c.py, c11 - c01, c01);
    return fmaf(c.pz, c1 - c0, c0);
}

// NEXT-2 / eq. 4: energy by eq. 2 from the score channel, gradient = the three per-vertex gradient
// channels interpolated with the same weights.  `cell` = packed entry of the score channel; the gradient channels sit
// chan_stride entries apart.
__device__ __forceinline__ float trilinear_eq4(const DevGrid &G, const CellRef &c, const Cell8 *cell,
                                               const float4 q0, const float4 q1, float &e_wall,
                                               float &gx, float &gy, float &gz)
{
    float4 a0, a1, b0, b1, d0, d1;
    ldg_cell(cell + (size_t)G.chan_stride, a0, a1);
    ldg_cell(cell + 2 * (size_t)G.chan_stride, b0, b1);
    ldg_cell(cell + 3 * (size_t)G.chan_stride, d0, d1);
    const float e = trilerp(c, q0, q1);
    apply_wall(G, c, trilerp(c, a0, a1), trilerp(c, b0, b1), trilerp(c, d0, d1), e_wall, gx, gy, gz);
    return e;
}

// Trilinear energy (eq. 2) and the gradient of the interpolant (eq. 3) from the two packed entries
// q0 (plane iz) and q1 (plane iz+1); clamped axes get zero grid gradient and the quadratic wall
// (reading S7).  Returns e_grid; adds to e_wall; gradient in kcal/mol/A.
__device__ __forceinline__ float trilinear(const DevGrid &G, const CellRef &c,
                                           const float4 q0, const float4 q1, float &e_wall,
                                           float &gx, float &gy, float &gz)
{
    const float d00 = q0.y - q0.x, d10 = q0.w - q0.z, d01 = q1.y - q1.x, d11 = q1.w - q1.z;
    const float c00 = fmaf(c.px, d00, q0.x), c10 = fmaf(c.px, d10, q0.z);
    const float c01 = fmaf(c.px, d01, q1.x), c11 = fmaf(c.px, d11, q1.z);
    const float dy0 = c10 - c00, dy1 = c11 - c01;
    const float c0 = fmaf(c.py, dy0, c00), c1 = fmaf(c.py, dy1, c01);
    const float dz = c1 - c0;
    const float e = fmaf(c.pz, dz, c0);                                               // eq. 2
    const float dx0 = fmaf(c.py, d10 - d00, d00), dx1 = fmaf(c.py, d11 - d01, d01);
    float ggx = fmaf(c.pz, dx1 - dx0, dx0) * G.inv_h;                                 // eq. 3, x
    float ggy = fmaf(c.pz, dy1 - dy0, dy0) * G.inv_h;                                 // eq. 3, y
    float ggz = dz * G.inv_h;                                                         // eq. 3, z
    apply_wall(G, c, ggx, ggy, ggz, e_wall, gx, gy, gz);
    return e;
}
