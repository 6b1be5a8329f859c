// search.cu -- A6 BFGS local optimizer, A7 many-copy Monte-Carlo, A8 top-k + RMSD clustering, all
// on the device (SURVEY.md 8(a) A6-A8, 8(c) O8-O10 and R-rules).
//
// One warp owns one copy for the whole search: pose, gradient, BFGS inverse Hessian and all
// optimizer vectors live in that warp's shared memory; the MC loop, the line search and the
// Metropolis test never leave the kernel.  Randomness is stateless Philox4x32-10 with
// counter = (copy, step, slot, system), so any step can be replayed alone.  Scalar reductions that
// feed a decision (g.p, y.s, norms, Armijo, Metropolis) are accumulated / compared in fp64.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <mutex>
#include <vector>

#include "common.cuh"
#include "eval_warp.cuh"
#include "host_compile.cuh"

namespace {

constexpr int SEARCH_WARPS = 4;
constexpr float PI_F = 3.14159265358979323846f;

struct OptBuf {
    float *x, *xt, *g, *gt, *d, *y, *hy, *H, *scratch;
};

__host__ __device__ inline int pad4(int v) { return (v + 3) & ~3; }

// floats of shared memory one warp needs for optimisation (excluding cur/best kept by the MC loop)
__host__ __device__ inline int opt_floats(int T, int n_pad)
{
    const int n = 6 + T, np_ = 7 + T;
    return 2 * pad4(np_) + 5 * pad4(n) + pad4(n * n) + 8 * n_pad + 2 * pad4(T) + 40 * T;
}

__device__ __forceinline__ OptBuf carve(float *base, int T, int n_pad)
{
    const int n = 6 + T, np_ = 7 + T;
    OptBuf b;
    b.x = base;               base += pad4(np_);
    b.xt = base;              base += pad4(np_);
    b.g = base;               base += pad4(n);
    b.gt = base;              base += pad4(n);
    b.d = base;               base += pad4(n);
    b.y = base;               base += pad4(n);
    b.hy = base;              base += pad4(n);
    b.H = base;               base += pad4(n * n);
    b.scratch = base;
    (void)n_pad;
    return b;
}

__device__ __forceinline__ void quat_mul_norm(float aw, float ax, float ay, float az,
                                              float bw, float bx, float by, float bz, float *out)
{
    float w = aw * bw - ax * bx - ay * by - az * bz;
    float x = aw * bx + ax * bw + ay * bz - az * by;
    float y = aw * by - ax * bz + ay * bw + az * bx;
    float z = aw * bz + ax * by - ay * bx + az * bw;
    const float inv = 1.0f / sqrtf(w * w + x * x + y * y + z * z);
    out[0] = w * inv; out[1] = x * inv; out[2] = y * inv; out[3] = z * inv;
}

// q <- normalize(quat(rotation vector w) (x) q)   (left-multiplied, lab frame)
__device__ __forceinline__ void rotate_quat(float wx, float wy, float wz, const float *q, float *out)
{
    const float phi = sqrtf(wx * wx + wy * wy + wz * wz);
    float qw, s;
    if (phi < 1e-6f) { qw = 1.0f; s = 0.5f; }
    else {
        float sn, cs;
        sincosf(0.5f * phi, &sn, &cs);
        qw = cs; s = sn / phi;
    }
    float ax = s * wx, ay = s * wy, az = s * wz;
    const float inv = 1.0f / sqrtf(qw * qw + ax * ax + ay * ay + az * az);
    quat_mul_norm(qw * inv, ax * inv, ay * inv, az * inv, q[0], q[1], q[2], q[3], out);
}

// out = x (+) alpha*d : t += s[0:3]; q <- normalize(quat(s[3:6]) (x) q); theta += s[6:]
__device__ __forceinline__ void pose_add_warp(int T, const float *x, const float *d, float alpha, float *out)
{
    const int lane = threadIdx.x & 31;
    if (lane < 3) out[lane] = fmaf(alpha, d[lane], x[lane]);
    if (lane == 3) rotate_quat(alpha * d[3], alpha * d[4], alpha * d[5], x + 3, out + 3);
    for (int k = lane; k < T; k += 32) out[7 + k] = fmaf(alpha, d[6 + k], x[7 + k]);
    __syncwarp();
}

__device__ __forceinline__ void set_identity(float *H, int n, float diag)
{
    const int lane = threadIdx.x & 31;
    for (int k = lane; k < n * n; k += 32) H[k] = (k / n == k % n) ? diag : 0.0f;
    __syncwarp();
}

#include "search_cta.cuh"

// O8: BFGS with backtracking.  b.x holds the start pose (quaternion normalised here) and the result.
// Written as one loop around a SINGLE evaluation site (the start pose is "trial" INIT), so that the evaluator and
// this routine inline into the kernels once: the compiler then sees that every buffer is shared memory and keeps
// P, G, L in registers / the constant bank instead of local memory (profiles/r1g.md).
// TRACE: one record per iteration started goes to `itrace` (layout: dock.h, DOCK_ITER_HEADER) -- the state the
// iteration starts from (pose, inverse Hessian) and its decision scalars, enough for the oracle to redo that one
// iteration from the same state (iteration-level teacher-forced parity).
template <bool EQ4, bool VEC4, bool TRACE = false>
__device__ __forceinline__ float local_opt_warp(const DevParams &P, const DevGrid &G, const DevLigand &L,
                                                const OptBuf &b, int cap, int &iters, int &evals, int &why,
                                                float *itrace = nullptr, int itrace_cap = 0)
{
    const int lane = threadIdx.x & 31;
    const int T = L.T, n = 6 + T, np_ = 7 + T;
    const int istride = DOCK_ITER_HEADER + np_ + n + n * n;
    why = DOCK_EXIT_CAP;
    if (lane == 0) {
        const float w = b.x[3], x = b.x[4], y = b.x[5], z = b.x[6];
        const float n2 = w * w + x * x + y * y + z * z;
        if (n2 > 0.f) { const float inv = 1.0f / sqrtf(n2); b.x[3] = w * inv; b.x[4] = x * inv; b.x[5] = y * inv; b.x[6] = z * inv; }
        else { b.x[3] = 1.f; b.x[4] = b.x[5] = b.x[6] = 0.f; }
    }
    __syncwarp();
    for (int k = lane; k < np_; k += 32) b.xt[k] = b.x[k];
    __syncwarp();
    float f = 0.0f, alpha = 1.0f, f_best = 0.0f;
    double gp = 0.0;
    bool init = true, fresh = true;
    const bool bb = P.optimizer == 1;          // Barzilai-Borwein (reading S13): no H, no line search;
    float *const x_best = b.H;                 // the best point seen is kept in the (unused) H buffer
    int it = 0, trial = 0;
    evals = 0;
    for (;;) {
        const float ft = eval_pose_warp<true, EQ4, VEC4>(P, G, L, b.xt, b.gt, b.scratch, nullptr);
        ++evals;
        if (init) {
            init = false;
            f = ft;
            for (int r = lane; r < n; r += 32) b.g[r] = b.gt[r];
            if (bb) {
                f_best = f;
                for (int k = lane; k < np_; k += 32) x_best[k] = b.x[k];
                __syncwarp();
            } else set_identity(b.H, n, 1.0f);
        } else if (bb) {                           // every BB step is taken: s = alpha d, y = g_new - g
            for (int r = lane; r < n; r += 32) {
                b.d[r] = alpha * b.d[r];
                b.y[r] = b.gt[r] - b.g[r];
                b.g[r] = b.gt[r];
            }
            for (int k = lane; k < np_; k += 32) b.x[k] = b.xt[k];
            f = ft;
            if (f < f_best) {
                f_best = f;
                for (int k = lane; k < np_; k += 32) x_best[k] = b.xt[k];
            }
            __syncwarp();
            if (TRACE && it < itrace_cap && lane == 0) itrace[(size_t)it * istride + 5] = ft;
            ++it;
        } else if ((double)ft - (double)f <= (double)P.c1 * (double)alpha * gp) {   // Armijo: accept the step
            double ys = 0.0, yy = 0.0, ss = 0.0;
            for (int r = lane; r < n; r += 32) {
                const float s = alpha * b.d[r], yv = b.gt[r] - b.g[r];
                b.d[r] = s;                        // d now holds s
                b.y[r] = yv;
                ys += (double)yv * (double)s; yy += (double)yv * (double)yv; ss += (double)s * (double)s;
            }
            ys = warp_sum_d(ys); yy = warp_sum_d(yy); ss = warp_sum_d(ss);
            for (int k = lane; k < np_; k += 32) b.x[k] = b.xt[k];
            for (int r = lane; r < n; r += 32) b.g[r] = b.gt[r];
            f = ft;
            __syncwarp();
            const bool upd = ys > (double)P.curv_eps * sqrt(ss) * sqrt(yy);
            if (upd) {
                if (fresh) { set_identity(b.H, n, (float)(ys / yy)); fresh = false; }
                for (int r = lane; r < n; r += 32) {
                    float a = 0.0f;
                    for (int c = 0; c < n; ++c) a = fmaf(b.H[r * n + c], b.y[c], a);
                    b.hy[r] = a;
                }
                __syncwarp();
                double acc = 0.0;
                for (int r = lane; r < n; r += 32) acc += (double)b.y[r] * (double)b.hy[r];
                const double yhy = warp_sum_d(acc);
                const double rho_d = 1.0 / ys;
                const float rho = (float)rho_d, coef = (float)(rho_d * rho_d * yhy + rho_d);
                // H <- (I - rho s y^T) H (I - rho y s^T) + rho s s^T, expanded for symmetric H
                for (int r = lane; r < n; r += 32) {
                    const float sr = b.d[r], hr = b.hy[r];
                    for (int c = 0; c < n; ++c) {
                        const float sc = b.d[c], hc = b.hy[c];
                        b.H[r * n + c] += fmaf(coef * sr, sc, -rho * fmaf(sr, hc, hr * sc));
                    }
                }
                __syncwarp();
            }
            if (TRACE && it < itrace_cap && lane == 0) {
                float *rec = itrace + (size_t)it * istride;
                rec[4] = alpha; rec[5] = f; rec[7] = (float)(trial + 1); rec[8] = upd ? 1.f : 0.f; rec[11] = fresh ? 1.f : 0.f;
            }
            ++it;
        } else {                                   // backtrack
            if (++trial >= P.max_trials) {         // no acceptable trial: stop
                why = DOCK_EXIT_LINESEARCH;
                if (TRACE && it < itrace_cap && lane == 0) {
                    float *rec = itrace + (size_t)it * istride;
                    rec[4] = alpha; rec[5] = ft; rec[6] = (float)DOCK_EXIT_LINESEARCH; rec[7] = (float)trial; rec[11] = fresh ? 1.f : 0.f;
                }
                break;
            }
            alpha *= P.shrink;
            pose_add_warp(T, b.x, b.d, alpha, b.xt);
            continue;
        }
        // ---- start iteration `it` ----
        if (it >= cap) break;
        double acc = 0.0;
        for (int r = lane; r < n; r += 32) acc += (double)b.g[r] * (double)b.g[r];
        const double gn2 = warp_sum_d(acc);
        if (TRACE && it < itrace_cap) {            // the state this iteration starts from
            float *rec = itrace + (size_t)it * istride;
            if (lane == 0) {
                rec[0] = f; rec[1] = (float)sqrt(gn2); rec[2] = rec[3] = rec[4] = rec[5] = 0.f;
                rec[6] = 0.f; rec[7] = 0.f; rec[8] = 0.f; rec[9] = 0.f; rec[10] = fresh ? 1.f : 0.f; rec[11] = fresh ? 1.f : 0.f;
            }
            for (int k = lane; k < np_; k += 32) rec[DOCK_ITER_HEADER + k] = b.x[k];
            for (int k = lane; k < n; k += 32) rec[DOCK_ITER_HEADER + np_ + k] = b.g[k];
            if (bb)                                // Barzilai-Borwein: the previous step (s, y) takes the place of H
                for (int k = lane; k < n; k += 32) {
                    rec[DOCK_ITER_HEADER + np_ + n + k] = it > 0 ? b.d[k] : 0.f;
                    rec[DOCK_ITER_HEADER + np_ + 2 * n + k] = it > 0 ? b.y[k] : 0.f;
                }
            else
                for (int k = lane; k < n * n; k += 32) rec[DOCK_ITER_HEADER + np_ + n + k] = b.H[k];
        }
        if (sqrt(gn2) < (double)P.gtol) {
            why = DOCK_EXIT_GTOL;
            if (TRACE && it < itrace_cap && lane == 0) itrace[(size_t)it * istride + 6] = (float)DOCK_EXIT_GTOL;
            break;
        }
        if (bb) {
            const double gnorm = sqrt(gn2);
            double al;
            int branch = 0;
            if (it == 0) al = (double)P.bb_step / gnorm;
            else {
                double sy = 0.0, ss = 0.0, yy = 0.0;
                for (int r = lane; r < n; r += 32) {
                    const double sv = (double)b.d[r], yv = (double)b.y[r];
                    sy += sv * yv; ss += sv * sv; yy += yv * yv;
                }
                sy = warp_sum_d(sy); ss = warp_sum_d(ss); yy = warp_sum_d(yy);
                branch = (sy > (double)P.curv_eps * sqrt(ss) * sqrt(yy)) ? 1 : 2;
                al = branch == 1 ? ss / sy : (double)P.bb_fallback / gnorm;
            }
            const bool capped = al * gnorm > (double)P.bb_step;
            if (capped) al = (double)P.bb_step / gnorm;
            alpha = (float)al;
            if (TRACE && it < itrace_cap && lane == 0) {
                float *rec = itrace + (size_t)it * istride;
                rec[4] = alpha; rec[7] = (float)branch; rec[9] = capped ? 1.f : 0.f;
            }
            __syncwarp();
            for (int r = lane; r < n; r += 32) b.d[r] = -b.g[r];
            __syncwarp();
            pose_add_warp(T, b.x, b.d, alpha, b.xt);
            continue;
        }
        for (int r = lane; r < n; r += 32) {
            float a = 0.0f;
            for (int c = 0; c < n; ++c) a = fmaf(b.H[r * n + c], b.g[c], a);
            b.d[r] = -a;
        }
        __syncwarp();
        acc = 0.0;
        for (int r = lane; r < n; r += 32) acc += (double)b.g[r] * (double)b.d[r];
        gp = warp_sum_d(acc);
        if (gp >= 0.0) {                           // not a descent direction: reset H = I
            set_identity(b.H, n, 1.0f);
            fresh = true;
            for (int r = lane; r < n; r += 32) b.d[r] = -b.g[r];
            __syncwarp();
            gp = -gn2;
            if (TRACE && it < itrace_cap && lane == 0) itrace[(size_t)it * istride + 9] = 1.f;
        }
        alpha = 1.0f;
        if (fresh) {
            acc = 0.0;
            for (int r = lane; r < n; r += 32) acc += (double)b.d[r] * (double)b.d[r];
            const double dn = sqrt(warp_sum_d(acc));
            if (dn > 1.0) alpha = (float)(1.0 / dn);
        }
        if (TRACE && it < itrace_cap && lane == 0) {
            float *rec = itrace + (size_t)it * istride;
            rec[2] = (float)gp; rec[3] = alpha;
        }
        trial = 0;
        pose_add_warp(T, b.x, b.d, alpha, b.xt);
    }
    if (bb) {                                      // non-monotone method: report the best point seen
        __syncwarp();
        for (int k = lane; k < np_; k += 32) b.x[k] = x_best[k];
        __syncwarp();
        f = f_best;
    }
    iters = it;
    return f;
}

// ---- local optimisation of a batch of poses (level-2 parity entry point) -------------------------
template <bool EQ4, bool VEC4, bool TRACE>
__global__ void __launch_bounds__(SEARCH_WARPS * 32)
local_opt_kernel(DevParams P, DevGrid G, DevLigand L, long long n_poses, int cap, int warp_floats,
                 const float *__restrict__ poses, float *__restrict__ out_pose, float *__restrict__ out_e,
                 int *__restrict__ out_iters, float *__restrict__ itrace, int itrace_cap)
{
    extern __shared__ float smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const long long p = (long long)blockIdx.x * SEARCH_WARPS + warp;
    if (p >= n_poses) return;
    const int np_ = 7 + L.T;
    const OptBuf b = carve(smem + (size_t)warp * warp_floats, L.T, L.n_pad);
    for (int k = lane; k < np_; k += 32) b.x[k] = poses[p * np_ + k];
    __syncwarp();
    int iters, evals, why;
    const size_t istride = DOCK_ITER_HEADER + np_ + (size_t)(6 + L.T) * (7 + L.T);
    const float e = local_opt_warp<EQ4, VEC4, TRACE>(P, G, L, b, cap, iters, evals, why,
                                                     TRACE ? itrace + (size_t)p * itrace_cap * istride : nullptr, itrace_cap);
    for (int k = lane; k < np_; k += 32) out_pose[p * np_ + k] = b.x[k];
    if (lane == 0) {
        out_e[p] = e;
        if (out_iters) { out_iters[3 * p] = iters; out_iters[3 * p + 1] = evals; out_iters[3 * p + 2] = why; }
    }
}

// ---- A7 Monte-Carlo ------------------------------------------------------------------------------
__device__ __forceinline__ float u24(uint32_t r) { return (float)(r >> 8) * (1.0f / 16777216.0f); }

// 4 CTAs per SM = 128 registers, no spills: 16 resident warps for the screening batches (143 vs 126 M evals/s on a
// 64-system config-3 slice), same latency for the 384-copy case (profiles/r1i.md)
template <bool EQ4, bool VEC4>
__global__ void __launch_bounds__(SEARCH_WARPS * 32, 4)
search_kernel(DevParams P, const DevSystem *__restrict__ systems, int n_systems, int copies, int steps,
              int cap, uint32_t seed_lo, uint32_t seed_hi, uint32_t sys_base, uint32_t copy_base, int t_max, int warp_floats,
              const float *__restrict__ init, float *__restrict__ best_pose, float *__restrict__ best_e,
              float *__restrict__ trace, unsigned long long *__restrict__ eval_counter)
{
    extern __shared__ float smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const long long gw = (long long)blockIdx.x * SEARCH_WARPS + warp;
    if (gw >= (long long)n_systems * copies) return;
    const uint32_t sys = (uint32_t)(gw / copies);
    const uint32_t copy = copy_base + (uint32_t)(gw % copies), psys = sys_base + sys;   // Philox counter words (R-rules)
    const DevGrid G = systems[sys].grid;
    const DevLigand L = systems[sys].lig;
    const int T = L.T, np_ = 7 + T, row = 7 + t_max;
    float *base = smem + (size_t)warp * warp_floats;
    float *cur = base, *best = base + pad4(row);
    const OptBuf b = carve(base + 2 * pad4(row), T, L.n_pad);

    int iters, evals, why;
    unsigned long long total_evals = 0;
    float e_cur = 0.0f, e_best = 0.0f;
    // step -1 = local optimisation of the initial pose (reading S16); one call site of the optimizer
    for (int step = -1; step < steps; ++step) {
        uint32_t r[4] = {0u, 0u, 0u, 0u};
        int kind = 0;
        if (step < 0) {
            for (int k = lane; k < np_; k += 32) b.x[k] = init[gw * row + k];
            __syncwarp();
        } else {
            philox4x32_10(copy, (uint32_t)step, 0u, psys, seed_lo, seed_hi, r);
            const uint32_t K = T > 0 ? 3u : 2u;
            kind = (int)__umulhi(r[0], K);
            for (int k = lane; k < np_; k += 32) b.x[k] = cur[k];
            __syncwarp();
            if (lane == 0) {
                if (kind == 0) {
                    for (int c = 0; c < 3; ++c) b.x[c] = cur[c] + P.amp_trans * (2.0f * u24(r[1 + c]) - 1.0f);
                } else if (kind == 1) {
                    rotate_quat(P.amp_rot * (2.0f * u24(r[1]) - 1.0f), P.amp_rot * (2.0f * u24(r[2]) - 1.0f),
                                P.amp_rot * (2.0f * u24(r[3]) - 1.0f), cur + 3, b.x + 3);
                } else {
                    const int k = (int)__umulhi(r[1], (uint32_t)T);
                    b.x[7 + k] = PI_F * (2.0f * u24(r[2]) - 1.0f);
                }
            }
            __syncwarp();
        }
        const float e_c = local_opt_warp<EQ4, VEC4>(P, G, L, b, cap, iters, evals, why);
        total_evals += evals;
        if (step < 0) {
            e_cur = e_best = e_c;
            for (int k = lane; k < np_; k += 32) { cur[k] = b.x[k]; best[k] = b.x[k]; }
            __syncwarp();
            continue;
        }
        uint32_t ra[4];
        philox4x32_10(copy, (uint32_t)step, 1u, psys, seed_lo, seed_hi, ra);
        const float u = u24(ra[0]);
        const bool accept = (e_c < e_cur) || ((double)u < exp(((double)e_cur - (double)e_c) / (double)P.t_mc));
        if (trace) {
            float *rec = trace + ((size_t)gw * steps + step) * (size_t)(DOCK_TRACE_HEADER + row);
            if (lane == 0) {
                rec[0] = e_cur; rec[1] = e_c; rec[2] = u; rec[3] = accept ? 1.0f : 0.0f;
                rec[4] = (float)iters; rec[5] = (float)evals; rec[6] = (float)kind; rec[7] = 0.0f;
            }
            for (int k = lane; k < row; k += 32) rec[DOCK_TRACE_HEADER + k] = k < np_ ? cur[k] : 0.0f;
            __syncwarp();
        }
        if (accept) {
            for (int k = lane; k < np_; k += 32) cur[k] = b.x[k];
            e_cur = e_c;
        }
        if (e_cur < e_best) {
            e_best = e_cur;
            for (int k = lane; k < np_; k += 32) best[k] = accept ? b.x[k] : cur[k];
        }
        __syncwarp();
    }
    for (int k = lane; k < row; k += 32) best_pose[gw * row + k] = k < np_ ? best[k] : 0.0f;
    if (lane == 0) {
        best_e[gw] = e_best;
        if (eval_counter) atomicAdd(eval_counter, total_evals);
    }
}

// ---- the same two kernels with one CTA of CTA_WARPS warps per pose / copy: speculative line search (search_cta.cuh) ----
template <bool EQ4, bool VEC4, bool TRACE>
__global__ void __launch_bounds__(CTA_THREADS, 3)
local_opt_cta_kernel(DevParams P, DevGrid G, DevLigand L, long long n_poses, int cap,
                     const float *__restrict__ poses, float *__restrict__ out_pose, float *__restrict__ out_e,
                     int *__restrict__ out_iters, float *__restrict__ itrace, int itrace_cap)
{
    extern __shared__ float smem[];
    const long long p = blockIdx.x;
    const int tid = threadIdx.x, np_ = 7 + L.T;
    const SpecBuf b = spec_carve(smem, L.T, L.n_pad);
    if (tid < np_) b.x[tid] = poses[p * np_ + tid];
    __syncthreads();
    int iters, evals, why;
    const size_t istride = DOCK_ITER_HEADER + np_ + (size_t)(6 + L.T) * (7 + L.T);
    const float e = local_opt_spec<EQ4, VEC4, TRACE>(P, G, L, b, cap, iters, evals, why,
                                                     TRACE ? itrace + (size_t)p * itrace_cap * istride : nullptr, itrace_cap);
    if (tid < np_) out_pose[p * np_ + tid] = b.x[tid];
    if (tid == 0) {
        out_e[p] = e;
        if (out_iters) { out_iters[3 * p] = iters; out_iters[3 * p + 1] = evals; out_iters[3 * p + 2] = why; }
    }
}

// 3 CTAs per SM (<= 168 registers): 444 copies resident on 148 SMs, so the paper's 384 copies run in one wave
template <bool EQ4, bool VEC4>
__global__ void __launch_bounds__(CTA_THREADS, 3)
search_cta_kernel(DevParams P, const DevSystem *__restrict__ systems, int n_systems, int copies, int steps,
                  int cap, uint32_t seed_lo, uint32_t seed_hi, uint32_t sys_base, uint32_t copy_base, int t_max,
                  const float *__restrict__ init, float *__restrict__ best_pose, float *__restrict__ best_e,
                  float *__restrict__ trace, unsigned long long *__restrict__ eval_counter)
{
    extern __shared__ float smem[];
    const int tid = threadIdx.x;
    const long long gw = blockIdx.x;
    const uint32_t sys = (uint32_t)(gw / copies);
    const uint32_t copy = copy_base + (uint32_t)(gw % copies), psys = sys_base + sys;
    const DevGrid G = systems[sys].grid;
    const DevLigand L = systems[sys].lig;
    const int T = L.T, np_ = 7 + T, row = 7 + t_max;
    float *cur = smem, *best = smem + pad4(row);
    const SpecBuf b = spec_carve(smem + 2 * pad4(row), T, L.n_pad);

    int iters, evals, why;
    unsigned long long total_evals = 0;
    float e_cur = 0.0f, e_best = 0.0f;
    for (int step = -1; step < steps; ++step) {
        uint32_t r[4] = {0u, 0u, 0u, 0u};
        int kind = 0;
        if (step < 0) {
            if (tid < np_) b.x[tid] = init[gw * row + tid];
            __syncthreads();
        } else {
            philox4x32_10(copy, (uint32_t)step, 0u, psys, seed_lo, seed_hi, r);
            const uint32_t K = T > 0 ? 3u : 2u;
            kind = (int)__umulhi(r[0], K);
            if (tid < np_) b.x[tid] = cur[tid];
            __syncthreads();
            if (tid == 0) {
                if (kind == 0) {
                    for (int c = 0; c < 3; ++c) b.x[c] = cur[c] + P.amp_trans * (2.0f * u24(r[1 + c]) - 1.0f);
                } else if (kind == 1) {
                    rotate_quat(P.amp_rot * (2.0f * u24(r[1]) - 1.0f), P.amp_rot * (2.0f * u24(r[2]) - 1.0f),
                                P.amp_rot * (2.0f * u24(r[3]) - 1.0f), cur + 3, b.x + 3);
                } else {
                    const int k = (int)__umulhi(r[1], (uint32_t)T);
                    b.x[7 + k] = PI_F * (2.0f * u24(r[2]) - 1.0f);
                }
            }
            __syncthreads();
        }
        const float e_c = local_opt_spec<EQ4, VEC4, false>(P, G, L, b, cap, iters, evals, why);
        total_evals += evals;
        if (step < 0) {
            e_cur = e_best = e_c;
            if (tid < np_) { cur[tid] = b.x[tid]; best[tid] = b.x[tid]; }
            __syncthreads();
            continue;
        }
        uint32_t ra[4];
        philox4x32_10(copy, (uint32_t)step, 1u, psys, seed_lo, seed_hi, ra);
        const float u = u24(ra[0]);
        const bool accept = (e_c < e_cur) || ((double)u < exp(((double)e_cur - (double)e_c) / (double)P.t_mc));
        if (trace) {
            float *rec = trace + ((size_t)gw * steps + step) * (size_t)(DOCK_TRACE_HEADER + row);
            if (tid == 0) {
                rec[0] = e_cur; rec[1] = e_c; rec[2] = u; rec[3] = accept ? 1.0f : 0.0f;
                rec[4] = (float)iters; rec[5] = (float)evals; rec[6] = (float)kind; rec[7] = 0.0f;
            }
            if (tid < row) rec[DOCK_TRACE_HEADER + tid] = tid < np_ ? cur[tid] : 0.0f;
        }
        __syncthreads();
        if (accept) {
            if (tid < np_) cur[tid] = b.x[tid];
            e_cur = e_c;
        }
        if (e_cur < e_best) {
            e_best = e_cur;
            if (tid < np_) best[tid] = accept ? b.x[tid] : cur[tid];
        }
        __syncthreads();
    }
    if (tid < row) best_pose[gw * row + tid] = tid < np_ ? best[tid] : 0.0f;
    if (tid == 0) {
        best_e[gw] = e_best;
        if (eval_counter) atomicAdd(eval_counter, total_evals);
    }
}

// ---- A8 top-k + greedy RMSD clustering -------------------------------------------------------------
// One CTA per system.  Bitonic sort of (E, copy) ascending with ties to the lower copy index, then
// warp 0 walks the ranking and keeps a pose iff its heavy-atom RMSD to every kept pose is >= rmsd_min.
__global__ void __launch_bounds__(256)
topk_kernel(const DevSystem *__restrict__ systems, int n, int n_pow2, int row, int k_max, float rmsd_min,
            const float *__restrict__ poses, const float *__restrict__ e,
            int *__restrict__ out_idx, int *__restrict__ out_count,
            float *__restrict__ out_pose, float *__restrict__ out_e)
{
    extern __shared__ float smem[];
    const int sys = blockIdx.x;
    const DevLigand L = systems[sys].lig;
    float *key = smem;                                  // [n_pow2]
    int *idx = reinterpret_cast<int *>(smem + n_pow2);  // [n_pow2]
    float *kept = smem + 2 * n_pow2;                    // [k_max][3*n_pad]
    float *cand = kept + (size_t)k_max * 3 * L.n_pad;   // [3*n_pad]
    float *sc = cand + 3 * L.n_pad;                     // sincos scratch
    float *pose_s = sc + 2 * pad4(L.T);                 // [row]
    const float *pe = e + (size_t)sys * n;
    const float *pp = poses + (size_t)sys * n * row;
    for (int i = threadIdx.x; i < n_pow2; i += blockDim.x) {
        float v = i < n ? pe[i] : INFINITY;
        if (v != v) v = INFINITY;                       // NaN ranks last
        key[i] = v;
        idx[i] = i < n ? i : 0x7fffffff;
    }
    __syncthreads();
    for (int size = 2; size <= n_pow2; size <<= 1)
        for (int stride = size >> 1; stride > 0; stride >>= 1) {
            for (int i = threadIdx.x; i < n_pow2; i += blockDim.x) {
                const int j = i ^ stride;
                if (j > i) {
                    const bool up = (i & size) == 0;
                    const float ki = key[i], kj = key[j];
                    const int ii = idx[i], ij = idx[j];
                    const bool i_after_j = (ki > kj) || (ki == kj && ii > ij);
                    if (i_after_j == up) { key[i] = kj; key[j] = ki; idx[i] = ij; idx[j] = ii; }
                }
            }
            __syncthreads();
        }
    if (threadIdx.x >= 32) return;
    const int lane = threadIdx.x, np = L.n_pad, N = L.N;
    const float thr = rmsd_min * rmsd_min * (float)N;
    int n_kept = 0;
    for (int rank = 0; rank < n && n_kept < k_max; ++rank) {
        const int c = idx[rank];
        for (int k = lane; k < 7 + L.T; k += 32) pose_s[k] = pp[(size_t)c * row + k];
        __syncwarp();
        pose_coords_warp(L, pose_s, cand, sc);
        bool ok = true;
        for (int m = 0; m < n_kept && ok; ++m) {
            const float *km = kept + (size_t)m * 3 * np;
            float s = 0.0f;
            for (int i = lane; i < N; i += 32) {
                const float dx = cand[i] - km[i], dy = cand[np + i] - km[np + i], dz = cand[2 * np + i] - km[2 * np + i];
                s += dx * dx + dy * dy + dz * dz;
            }
            s = warp_sum(s);
            if (s < thr) ok = false;
        }
        if (ok) {
            float *km = kept + (size_t)n_kept * 3 * np;
            for (int i = lane; i < 3 * np; i += 32) km[i] = cand[i];
            if (lane == 0) {
                out_idx[(size_t)sys * k_max + n_kept] = c;
                if (out_e) out_e[(size_t)sys * k_max + n_kept] = key[rank];
            }
            if (out_pose)
                for (int k = lane; k < row; k += 32) out_pose[((size_t)sys * k_max + n_kept) * row + k] = pp[(size_t)c * row + k];
            ++n_kept;
        }
        __syncwarp();
    }
    for (int m = n_kept + lane; m < k_max; m += 32) {
        out_idx[(size_t)sys * k_max + m] = -1;
        if (out_e) out_e[(size_t)sys * k_max + m] = 0.0f;
    }
    if (lane == 0) out_count[sys] = n_kept;
}

// dynamic shared memory of topk_kernel; the callers check it against the 200 KB limit BEFORE they enqueue anything
size_t topk_smem_bytes(int n_systems, const DevLigand *ligs_host, int n, int row, int k, int *n_pow2_out)
{
    int n_pow2 = 1;
    while (n_pow2 < n) n_pow2 <<= 1;
    int np_max = 0, t_max = 0;
    for (int s = 0; s < n_systems; ++s) {
        np_max = ligs_host[s].n_pad > np_max ? ligs_host[s].n_pad : np_max;
        t_max = ligs_host[s].T > t_max ? ligs_host[s].T : t_max;
    }
    if (n_pow2_out) *n_pow2_out = n_pow2;
    return sizeof(float) * ((size_t)2 * n_pow2 + (size_t)(k + 1) * 3 * np_max + 2 * pad4(t_max) + pad4(row) + 8);
}

int launch_topk(const DevSystem *systems_dev, int n_systems, const DevLigand *ligs_host, int n, int row, int k,
                float rmsd_min, const float *poses, const float *e, int *out_idx, int *out_count,
                float *out_pose, float *out_e, cudaStream_t stream)
{
    int n_pow2 = 1;
    const size_t smem = topk_smem_bytes(n_systems, ligs_host, n, row, k, &n_pow2);
    if (smem > 200 * 1024) return DOCK_EINVAL;
    if (smem > 48 * 1024)
        DOCK_CUDA_CHECK(cudaFuncSetAttribute(topk_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    topk_kernel<<<n_systems, 256, smem, stream>>>(systems_dev, n, n_pow2, row, k, rmsd_min, poses, e, out_idx, out_count, out_pose, out_e);
    DOCK_LAUNCH_CHECK();
    return DOCK_OK;
}

void host_init_pose(const dock_box *box, int T, uint64_t seed, uint32_t system, uint32_t copy, float *out)
{
    const uint32_t k0 = (uint32_t)(seed & 0xffffffffu), k1 = (uint32_t)(seed >> 32);
    const double two_pi = 6.283185307179586476925286766559, pi = 3.14159265358979323846;
    auto u = [](uint32_t r) { return (double)(r >> 8) * (1.0 / 16777216.0); };
    uint32_t r[4];
    philox4x32_10(copy, 0xffffffffu, 0u, system, k0, k1, r);
    for (int c = 0; c < 3; ++c)
        out[c] = (float)((double)box->center[c] - 0.5 * (double)box->size[c] + u(r[c]) * (double)box->size[c]);
    philox4x32_10(copy, 0xffffffffu, 1u, system, k0, k1, r);
    const double u1 = u(r[0]), u2 = u(r[1]), u3 = u(r[2]);
    out[3] = (float)(std::sqrt(u1) * std::cos(two_pi * u3));
    out[4] = (float)(std::sqrt(1.0 - u1) * std::sin(two_pi * u2));
    out[5] = (float)(std::sqrt(1.0 - u1) * std::cos(two_pi * u2));
    out[6] = (float)(std::sqrt(u1) * std::sin(two_pi * u3));
    for (int k = 0; k < T; ++k) {
        if (k % 4 == 0) philox4x32_10(copy, 0xffffffffu, 2u + (uint32_t)(k / 4), system, k0, k1, r);
        out[7 + k] = (float)(pi * (2.0 * u(r[k % 4]) - 1.0));
    }
}

}  // namespace

extern "C" int dock_init_poses(const dock_box *box, int32_t T, uint64_t seed, uint32_t system, uint32_t copy_base,
                               int32_t copies, float *out_host)
{
    if (!box || !out_host || T < 0 || T > DOCK_MAX_TORSIONS || copies < 0) return DOCK_EINVAL;
    for (int c = 0; c < copies; ++c) host_init_pose(box, T, seed, system, copy_base + (uint32_t)c, out_host + (size_t)c * (7 + T));
    return DOCK_OK;
}

// NEXT-3 (Fig. 3; reading S22): translation restrained to box (intersected with) the union of balls of
// `radius` around the predicted site points, by rejection from the Philox slots 0x100 + attempt (256 attempts,
// then the site point copy mod n_site); orientation and torsions as in dock_init_poses.
extern "C" int dock_init_poses_site(const dock_box *box, int32_t T, uint64_t seed, uint32_t system, uint32_t copy_base,
                                    int32_t copies, int32_t n_site, const float *site_xyz_host, float radius, float *out_host)
{
    if (!box || !out_host || T < 0 || T > DOCK_MAX_TORSIONS || copies < 0) return DOCK_EINVAL;
    if (n_site < 1 || !site_xyz_host || !(radius > 0.f)) return DOCK_EINVAL;
    const uint32_t k0 = (uint32_t)(seed & 0xffffffffu), k1 = (uint32_t)(seed >> 32);
    const double r2max = (double)radius * (double)radius;
    for (int ci = 0; ci < copies; ++ci) {
        const uint32_t c = copy_base + (uint32_t)ci;
        float *out = out_host + (size_t)ci * (7 + T);
        host_init_pose(box, T, seed, system, c, out);
        double t[3] = {0, 0, 0};
        bool found = false;
        for (int a = 0; a < 256 && !found; ++a) {
            uint32_t r[4];
            philox4x32_10(c, 0xffffffffu, 0x100u + (uint32_t)a, system, k0, k1, r);
            for (int d = 0; d < 3; ++d)
                t[d] = (double)box->center[d] - 0.5 * (double)box->size[d] + (double)(r[d] >> 8) * (1.0 / 16777216.0) * (double)box->size[d];
            for (int k = 0; k < n_site && !found; ++k) {
                const double dx = t[0] - (double)site_xyz_host[3 * k], dy = t[1] - (double)site_xyz_host[3 * k + 1],
                             dz = t[2] - (double)site_xyz_host[3 * k + 2];
                if (dx * dx + dy * dy + dz * dz <= r2max) found = true;
            }
        }
        if (!found)
            for (int d = 0; d < 3; ++d) t[d] = (double)site_xyz_host[3 * (c % (uint32_t)n_site) + d];
        for (int d = 0; d < 3; ++d) out[d] = (float)t[d];
    }
    return DOCK_OK;
}

namespace {
// dock_params.search_kernel: 1 = warp per copy, 2 = CTA of 4 warps per copy with the speculative line search, 0 = by size.
// Four warps per copy pay while the launch cannot fill the GPU with one warp per copy: up to CTA_AUTO_MAX copies in total
// (measured, profiles/r2c.md).  The two kernels give bit-identical results.
constexpr long long CTA_AUTO_MAX = 512;
bool use_cta_kernel(const dock_params *p, long long total_copies)
{
    if (p->search_kernel == 2) return true;
    if (p->search_kernel == 1) return false;
    return total_copies <= CTA_AUTO_MAX;       // BFGS: speculative line search; Barzilai-Borwein: the four warps share each evaluation
}

int local_opt_launch(const dock_params *params, const dock_grid *grid, const dock_ligand *ligand,
                     int64_t n_poses, int32_t max_iters, const float *poses_dev,
                     float *out_pose_dev, float *out_e_dev, int32_t *out_iters_dev,
                     float *iter_trace_dev, int32_t trace_cap,
                     void *ws_dev, size_t ws_bytes, size_t *needed, void *stream_)
{
    DevParams P;
    DevGrid G;
    LigandBlob blob;
    if (dock_make_dev_params(params, &P) != DOCK_OK || dock_make_dev_grid(params, grid, &G) != DOCK_OK) return DOCK_EINVAL;
    if (dock_compile_ligand(params, grid, ligand, blob) != DOCK_OK) return DOCK_EINVAL;
    if (n_poses < 0 || max_iters < 0 || trace_cap < 0) return DOCK_EINVAL;
    if (needed) *needed = blob.bytes.size();
    if (!ws_dev || ws_bytes < blob.bytes.size()) return DOCK_EWORKSPACE;
    if (n_poses == 0) return DOCK_OK;
    if (!poses_dev || !out_pose_dev || !out_e_dev) return DOCK_EINVAL;
    cudaStream_t stream = (cudaStream_t)stream_;
    DOCK_CUDA_CHECK(cudaMemcpyAsync(ws_dev, blob.bytes.data(), blob.bytes.size(), cudaMemcpyHostToDevice, stream));
    const DevLigand L = dock_relocate_ligand(blob, (const unsigned char *)ws_dev);
    const bool eq4 = G.channels == 4, tr = iter_trace_dev != nullptr;
    if (use_cta_kernel(params, n_poses)) {
        const size_t smem_c = (size_t)spec_floats(L.T, L.n_pad) * sizeof(float);
        if (smem_c > 200 * 1024) return DOCK_EINVAL;
        if (n_poses > 0x7fffffffLL) return DOCK_EINVAL;
        const bool v4 = L.N <= 48;
        auto kc = tr ? (eq4 ? (v4 ? local_opt_cta_kernel<true, true, true> : local_opt_cta_kernel<true, false, true>)
                            : (v4 ? local_opt_cta_kernel<false, true, true> : local_opt_cta_kernel<false, false, true>))
                     : (eq4 ? (v4 ? local_opt_cta_kernel<true, true, false> : local_opt_cta_kernel<true, false, false>)
                            : (v4 ? local_opt_cta_kernel<false, true, false> : local_opt_cta_kernel<false, false, false>));
        if (smem_c > 48 * 1024)
            DOCK_CUDA_CHECK(cudaFuncSetAttribute(kc, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_c));
        kc<<<(unsigned)n_poses, CTA_THREADS, smem_c, stream>>>(P, G, L, n_poses, max_iters, poses_dev, out_pose_dev, out_e_dev,
                                                              out_iters_dev, iter_trace_dev, trace_cap);
        DOCK_LAUNCH_CHECK();
        return DOCK_OK;
    }
    const int warp_floats = opt_floats(L.T, L.n_pad);
    const size_t smem = (size_t)SEARCH_WARPS * warp_floats * sizeof(float);
    if (smem > 200 * 1024) return DOCK_EINVAL;
    // shared-memory layout of the evaluator (eval_warp.cuh): float4 per atom unless the ligand is large
    const bool vec4 = L.N <= 48;
    auto kern = tr ? (eq4 ? (vec4 ? local_opt_kernel<true, true, true> : local_opt_kernel<true, false, true>)
                          : (vec4 ? local_opt_kernel<false, true, true> : local_opt_kernel<false, false, true>))
                   : (eq4 ? (vec4 ? local_opt_kernel<true, true, false> : local_opt_kernel<true, false, false>)
                          : (vec4 ? local_opt_kernel<false, true, false> : local_opt_kernel<false, false, false>));
    if (smem > 48 * 1024)
        DOCK_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const unsigned blocks = (unsigned)((n_poses + SEARCH_WARPS - 1) / SEARCH_WARPS);
    kern<<<blocks, SEARCH_WARPS * 32, smem, stream>>>(P, G, L, n_poses, max_iters, warp_floats, poses_dev,
                                                     out_pose_dev, out_e_dev, out_iters_dev, iter_trace_dev, trace_cap);
    DOCK_LAUNCH_CHECK();
    return DOCK_OK;
}
}  // namespace

extern "C" int dock_local_opt_batch(const dock_params *params, const dock_grid *grid, const dock_ligand *ligand,
                                    int64_t n_poses, int32_t max_iters, const float *poses_dev,
                                    float *out_pose_dev, float *out_e_dev, int32_t *out_iters_dev,
                                    void *ws_dev, size_t ws_bytes, size_t *needed, void *stream_)
{
    return local_opt_launch(params, grid, ligand, n_poses, max_iters, poses_dev, out_pose_dev, out_e_dev, out_iters_dev,
                            nullptr, 0, ws_dev, ws_bytes, needed, stream_);
}

extern "C" int dock_local_opt_trace(const dock_params *params, const dock_grid *grid, const dock_ligand *ligand,
                                    int64_t n_poses, int32_t max_iters, const float *poses_dev,
                                    float *out_pose_dev, float *out_e_dev, int32_t *out_iters_dev,
                                    float *iter_trace_dev, int32_t trace_cap,
                                    void *ws_dev, size_t ws_bytes, size_t *needed, void *stream_)
{
    if (!iter_trace_dev && ws_dev) return DOCK_EINVAL;
    return local_opt_launch(params, grid, ligand, n_poses, max_iters, poses_dev, out_pose_dev, out_e_dev, out_iters_dev,
                            iter_trace_dev, trace_cap, ws_dev, ws_bytes, needed, stream_);
}

extern "C" int dock_search(const dock_params *params, int32_t n_systems,
                           const dock_grid *grids, const dock_ligand *ligands, const dock_box *boxes,
                           int32_t copies, int32_t steps, int32_t bfgs_max_iters, uint64_t seed,
                           uint32_t system_base, uint32_t copy_base,
                           const float *init_poses_dev,
                           float *best_pose_dev, float *best_e_dev,
                           float *topk_pose_dev, float *topk_e_dev, int32_t *topk_idx_dev, int32_t *topk_count_dev,
                           float *trace_dev, uint64_t *eval_counter_dev,
                           void *ws_dev, size_t ws_bytes, size_t *needed, void *stream_)
{
    DevParams P;
    if (dock_make_dev_params(params, &P) != DOCK_OK) return DOCK_EINVAL;
    if (n_systems < 1 || !grids || !ligands || copies < 1 || steps < 0 || bfgs_max_iters < 0) return DOCK_EINVAL;
    if (!init_poses_dev && !boxes) return DOCK_EINVAL;
    std::vector<LigandBlob> blobs(n_systems);
    std::vector<DevSystem> sys(n_systems);
    int t_max = 0, wf_max = 0;
    size_t blob_bytes = 0;
    for (int s = 0; s < n_systems; ++s) {
        if (dock_make_dev_grid(params, &grids[s], &sys[s].grid) != DOCK_OK) return DOCK_EINVAL;
        if (dock_compile_ligand(params, &grids[s], &ligands[s], blobs[s]) != DOCK_OK) return DOCK_EINVAL;
        blob_bytes += blobs[s].bytes.size();
        t_max = ligands[s].T > t_max ? ligands[s].T : t_max;
    }
    const int row = 7 + t_max;
    for (int s = 0; s < n_systems; ++s) {
        const int wf = 2 * pad4(row) + opt_floats(ligands[s].T, blobs[s].rel.n_pad);
        wf_max = wf > wf_max ? wf : wf_max;
    }
    // everything that can be rejected is rejected here, before the workspace answer and before anything is enqueued
    const bool want_topk = topk_idx_dev || topk_count_dev || topk_pose_dev || topk_e_dev;
    if (want_topk && (!topk_idx_dev || !topk_count_dev)) return DOCK_EINVAL;
    for (int s2 = 1; s2 < n_systems; ++s2)
        if (sys[s2].grid.channels != sys[0].grid.channels) return DOCK_EINVAL;      // one gradient mode per launch
    const bool cta = use_cta_kernel(params, (long long)n_systems * copies);
    size_t smem = (size_t)SEARCH_WARPS * wf_max * sizeof(float);
    if (cta) {
        int cf_max = 0;
        for (int s2 = 0; s2 < n_systems; ++s2)
            cf_max = std::max(cf_max, 2 * pad4(row) + spec_floats(ligands[s2].T, blobs[s2].rel.n_pad));
        smem = (size_t)cf_max * sizeof(float);
    }
    if (smem > 200 * 1024) return DOCK_EINVAL;
    if (want_topk) {
        std::vector<DevLigand> rel(n_systems);
        for (int s2 = 0; s2 < n_systems; ++s2) rel[s2] = blobs[s2].rel;
        if (topk_smem_bytes(n_systems, rel.data(), copies, row, params->topk, nullptr) > 200 * 1024) return DOCK_EINVAL;
    }
    const size_t b_sys = align_up(sizeof(DevSystem) * n_systems, 256);
    const size_t b_init = init_poses_dev ? 0 : align_up((size_t)n_systems * copies * row * sizeof(float), 256);
    const size_t need = blob_bytes + b_sys + b_init;
    if (needed) *needed = need;
    if (!ws_dev || ws_bytes < need) return DOCK_EWORKSPACE;
    if (!best_pose_dev || !best_e_dev) return DOCK_EINVAL;

    cudaStream_t stream = (cudaStream_t)stream_;
    unsigned char *ws = (unsigned char *)ws_dev;
    std::vector<unsigned char> image(blob_bytes);
    std::vector<DevLigand> ligs(n_systems);
    size_t off = 0;
    for (int s = 0; s < n_systems; ++s) {
        std::memcpy(image.data() + off, blobs[s].bytes.data(), blobs[s].bytes.size());
        sys[s].lig = dock_relocate_ligand(blobs[s], ws + off);
        ligs[s] = sys[s].lig;
        if (boxes)
            for (int c = 0; c < 3; ++c) {
                sys[s].box_lo[c] = boxes[s].center[c] - 0.5f * boxes[s].size[c];
                sys[s].box_size[c] = boxes[s].size[c];
            }
        off += blobs[s].bytes.size();
    }
    DOCK_CUDA_CHECK(cudaMemcpyAsync(ws, image.data(), blob_bytes, cudaMemcpyHostToDevice, stream));
    DevSystem *sys_dev = (DevSystem *)(ws + blob_bytes);
    DOCK_CUDA_CHECK(cudaMemcpyAsync(sys_dev, sys.data(), sizeof(DevSystem) * n_systems, cudaMemcpyHostToDevice, stream));
    const float *init = init_poses_dev;
    if (!init) {
        std::vector<float> h((size_t)n_systems * copies * row, 0.0f);
        for (int s = 0; s < n_systems; ++s)
            for (int c = 0; c < copies; ++c)
                host_init_pose(&boxes[s], ligands[s].T, seed, system_base + (uint32_t)s, copy_base + (uint32_t)c,
                               h.data() + ((size_t)s * copies + c) * row);
        float *d = (float *)(ws + blob_bytes + b_sys);
        DOCK_CUDA_CHECK(cudaMemcpyAsync(d, h.data(), h.size() * sizeof(float), cudaMemcpyHostToDevice, stream));
        init = d;
    }
    const long long total = (long long)n_systems * copies;
    if (total > 0x7fffffffLL) return DOCK_EINVAL;
    int n_max = 0;
    for (int s2 = 0; s2 < n_systems; ++s2) n_max = std::max(n_max, (int)ligands[s2].N);
    const bool vec4 = n_max <= 48;        // float4 per atom unless the ligands are large (eval_warp.cuh)
    if (cta) {
        auto kc = sys[0].grid.channels == 4 ? (vec4 ? search_cta_kernel<true, true> : search_cta_kernel<true, false>)
                                            : (vec4 ? search_cta_kernel<false, true> : search_cta_kernel<false, false>);
        if (smem > 48 * 1024)
            DOCK_CUDA_CHECK(cudaFuncSetAttribute(kc, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        kc<<<(unsigned)total, CTA_THREADS, smem, stream>>>(
            P, sys_dev, n_systems, copies, steps, bfgs_max_iters, (uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32),
            system_base, copy_base, t_max, init, best_pose_dev, best_e_dev, trace_dev, (unsigned long long *)eval_counter_dev);
        DOCK_LAUNCH_CHECK();
    } else {
        auto kern = sys[0].grid.channels == 4 ? (vec4 ? search_kernel<true, true> : search_kernel<true, false>)
                                              : (vec4 ? search_kernel<false, true> : search_kernel<false, false>);
        if (smem > 48 * 1024)
            DOCK_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        const unsigned blocks = (unsigned)((total + SEARCH_WARPS - 1) / SEARCH_WARPS);
        kern<<<blocks, SEARCH_WARPS * 32, smem, stream>>>(
            P, sys_dev, n_systems, copies, steps, bfgs_max_iters, (uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32),
            system_base, copy_base, t_max, wf_max, init, best_pose_dev, best_e_dev, trace_dev, (unsigned long long *)eval_counter_dev);
        DOCK_LAUNCH_CHECK();
    }
    if (want_topk)
        return launch_topk(sys_dev, n_systems, ligs.data(), copies, row, params->topk, params->cluster_rmsd,
                           best_pose_dev, best_e_dev, topk_idx_dev, topk_count_dev, topk_pose_dev, topk_e_dev, stream);
    return DOCK_OK;
}

extern "C" int dock_topk(const dock_params *params, const dock_ligand *ligand, int32_t n,
                         const float *poses_dev, const float *e_dev,
                         int32_t *out_idx_dev, int32_t *out_count_dev,
                         void *ws_dev, size_t ws_bytes, size_t *needed, void *stream_)
{
    if (dock_validate_params(params) != DOCK_OK || !ligand || n < 0) return DOCK_EINVAL;
    LigandBlob blob;
    if (dock_compile_ligand(params, nullptr, ligand, blob) != DOCK_OK) return DOCK_EINVAL;
    const size_t need = blob.bytes.size() + align_up(sizeof(DevSystem), 256);
    if (needed) *needed = need;
    if (!ws_dev || ws_bytes < need) return DOCK_EWORKSPACE;
    if (!out_idx_dev || !out_count_dev || (n > 0 && (!poses_dev || !e_dev))) return DOCK_EINVAL;
    cudaStream_t stream = (cudaStream_t)stream_;
    unsigned char *ws = (unsigned char *)ws_dev;
    DOCK_CUDA_CHECK(cudaMemcpyAsync(ws, blob.bytes.data(), blob.bytes.size(), cudaMemcpyHostToDevice, stream));
    DevSystem sys;
    std::memset(&sys, 0, sizeof(sys));
    sys.lig = dock_relocate_ligand(blob, ws);
    DevSystem *sys_dev = (DevSystem *)(ws + blob.bytes.size());
    DOCK_CUDA_CHECK(cudaMemcpyAsync(sys_dev, &sys, sizeof(sys), cudaMemcpyHostToDevice, stream));
    return launch_topk(sys_dev, 1, &sys.lig, n, 7 + ligand->T, params->topk, params->cluster_rmsd, poses_dev, e_dev,
                       out_idx_dev, out_count_dev, nullptr, nullptr, stream);
}

extern "C" int dock_system_host(const dock_params *params, const dock_protein *protein, const dock_box *box,
                                const dock_ligand *ligand, int32_t n_lig_types, const int32_t *lig_types,
                                int32_t copies, int32_t steps, int32_t bfgs_max_iters, uint64_t seed,
                                float *out_topk_pose_host, float *out_topk_e_host, int32_t *out_count_host,
                                uint64_t *out_evals_host,
                                float *grid_dev, size_t grid_bytes, void *ws_dev, size_t ws_bytes, size_t *needed, void *stream_)
{
    if (!params || !protein || !box || !ligand || copies < 1) return DOCK_EINVAL;
    if (dock_validate_params(params) != DOCK_OK) return DOCK_EINVAL;
    int32_t dims[3];
    if (dock_grid_dims(box, dims) != DOCK_OK) return DOCK_EINVAL;
    const int k = params->topk, row = 7 + ligand->T;
    // outputs carved from the front of the workspace, then the sub-call workspaces
    const size_t b_best = align_up((size_t)copies * row * sizeof(float), 256);
    const size_t b_beste = align_up((size_t)copies * sizeof(float), 256);
    const size_t b_tp = align_up((size_t)k * row * sizeof(float), 256);
    const size_t b_te = align_up((size_t)k * sizeof(float), 256);
    const size_t b_ti = align_up((size_t)k * sizeof(int32_t), 256);
    const size_t b_misc = 256;   // count (int32) + eval counter (uint64 at +8)
    const size_t head = b_best + b_beste + b_tp + b_te + b_ti + b_misc;
    size_t need_grid = 0, need_search = 0;
    dock_grid desc;
    int rc = dock_build_grids(params, protein, box, n_lig_types, lig_types, nullptr, 0, nullptr, nullptr, 0, &need_grid, nullptr);
    if (rc != DOCK_EWORKSPACE) return rc == DOCK_OK ? DOCK_EINVAL : rc;
    // descriptor for the size query of the search
    std::memset(&desc, 0, sizeof(desc));
    for (int c = 0; c < 3; ++c) desc.dims[c] = dims[c];
    desc.spacing = box->spacing;
    desc.n_maps = n_lig_types;
    for (int t = 0; t < DOCK_MAX_XS_TYPES; ++t) desc.type_to_map[t] = -1;
    for (int m = 0; m < n_lig_types; ++m)
        if (lig_types[m] >= 0 && lig_types[m] < DOCK_MAX_XS_TYPES) desc.type_to_map[lig_types[m]] = m;
    desc.data_dev = grid_dev ? grid_dev : (const float *)256;
    desc.packed_dev = desc.data_dev;
    float dummy;
    rc = dock_search(params, 1, &desc, ligand, box, copies, steps, bfgs_max_iters, seed, 0u, 0u, nullptr, &dummy, &dummy,
                     nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, 0, &need_search, nullptr);
    if (rc != DOCK_EWORKSPACE) return rc == DOCK_OK ? DOCK_EINVAL : rc;
    const size_t need = head + align_up(need_grid, 256) + align_up(need_search, 256);
    if (needed) *needed = need;
    if (!ws_dev || ws_bytes < need) return DOCK_EWORKSPACE;
    if (!grid_dev || !out_topk_pose_host || !out_topk_e_host || !out_count_host) return DOCK_EINVAL;
    cudaStream_t stream = (cudaStream_t)stream_;
    unsigned char *ws = (unsigned char *)ws_dev;
    float *d_best = (float *)ws, *d_beste = (float *)(ws + b_best);
    float *d_tp = (float *)(ws + b_best + b_beste), *d_te = (float *)(ws + b_best + b_beste + b_tp);
    int32_t *d_ti = (int32_t *)(ws + b_best + b_beste + b_tp + b_te);
    int32_t *d_cnt = (int32_t *)(ws + head - b_misc);
    uint64_t *d_ev = (uint64_t *)(ws + head - b_misc + 8);
    unsigned char *ws_grid = ws + head, *ws_search = ws + head + align_up(need_grid, 256);
    DOCK_CUDA_CHECK(cudaMemsetAsync(d_cnt, 0, b_misc, stream));
    rc = dock_build_grids(params, protein, box, n_lig_types, lig_types, grid_dev, grid_bytes, &desc, ws_grid, need_grid, nullptr, stream_);
    if (rc != DOCK_OK) return rc;
    rc = dock_search(params, 1, &desc, ligand, box, copies, steps, bfgs_max_iters, seed, 0u, 0u, nullptr, d_best, d_beste,
                     d_tp, d_te, d_ti, d_cnt, nullptr, d_ev, ws_search, need_search, nullptr, stream_);
    if (rc != DOCK_OK) return rc;
    DOCK_CUDA_CHECK(cudaMemcpyAsync(out_topk_pose_host, d_tp, (size_t)k * row * sizeof(float), cudaMemcpyDeviceToHost, stream));
    DOCK_CUDA_CHECK(cudaMemcpyAsync(out_topk_e_host, d_te, (size_t)k * sizeof(float), cudaMemcpyDeviceToHost, stream));
    DOCK_CUDA_CHECK(cudaMemcpyAsync(out_count_host, d_cnt, sizeof(int32_t), cudaMemcpyDeviceToHost, stream));
    if (out_evals_host) DOCK_CUDA_CHECK(cudaMemcpyAsync(out_evals_host, d_ev, sizeof(uint64_t), cudaMemcpyDeviceToHost, stream));
    DOCK_CUDA_CHECK(cudaStreamSynchronize(stream));
    return DOCK_OK;
}

// ---- dock_topk_fixed: A8 for callers that cannot allocate device memory ------------------------
// dock_topk keeps the compiled ligand tables and the system descriptor its kernel reads in a workspace the caller
// allocates.  Some callers have no way to do that: code running where a cudaMalloc is illegal or would stall (inside
// another framework's stream-ordered region, a plug-in that was handed pointers but no allocator, a real-time loop
// that must not touch the driver's heap).  For them the same scratch lives in the array below, which is part of the
// loaded library image: DOCK_TOPK_FIXED_BYTES on EVERY device that loads libdock_b200.so, from load until exit.
//
// The array's name is only meaningful to device code.  On the host it is a shadow symbol, not a device address, so the
// launch path never passes it along: each device's real address is looked up once with cudaGetSymbolAddress (with that
// device current) and cached in g_topk_fixed_addr.
namespace {

static __device__ __align__(256) unsigned char g_topk_fixed_scratch[DOCK_TOPK_FIXED_BYTES];

constexpr int TOPK_FIXED_MAX_DEVICES = 64;
std::mutex g_topk_fixed_mu;
unsigned char *g_topk_fixed_addr[TOPK_FIXED_MAX_DEVICES];   // per device, nullptr until the first call on it

// Device address of the scratch array on the CURRENT device (looked up on the first call there, then cached).
int topk_fixed_scratch(unsigned char **out)
{
    int dev = -1;
    DOCK_CUDA_CHECK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= TOPK_FIXED_MAX_DEVICES) return DOCK_EINVAL;
    std::lock_guard<std::mutex> lock(g_topk_fixed_mu);
    if (!g_topk_fixed_addr[dev]) {
        void *p = nullptr;
        DOCK_CUDA_CHECK(cudaGetSymbolAddress(&p, g_topk_fixed_scratch));
        if (!p) return DOCK_ECUDA;
        g_topk_fixed_addr[dev] = (unsigned char *)p;
    }
    *out = g_topk_fixed_addr[dev];
    return DOCK_OK;
}

}  // namespace

extern "C" int dock_topk_fixed(const dock_params *params, const dock_ligand *ligand, int32_t n,
                               const float *poses_dev, const float *e_dev,
                               int32_t *out_idx_dev, int32_t *out_count_dev, size_t *needed, void *stream_)
{
    if (dock_validate_params(params) != DOCK_OK || !ligand || n < 0) return DOCK_EINVAL;
    LigandBlob blob;
    if (dock_compile_ligand(params, nullptr, ligand, blob) != DOCK_OK) return DOCK_EINVAL;
    const size_t need = blob.bytes.size() + align_up(sizeof(DevSystem), 256);      // same layout as dock_topk's workspace
    if (needed) *needed = need;
    if (need > (size_t)DOCK_TOPK_FIXED_BYTES) return DOCK_ECAPACITY;                // nothing enqueued, nothing written
    if (!out_idx_dev || !out_count_dev || (n > 0 && (!poses_dev || !e_dev))) return DOCK_EINVAL;
    DevSystem sys;
    std::memset(&sys, 0, sizeof(sys));
    sys.lig = blob.rel;                                                             // sizes only, for the shared-memory check
    if (topk_smem_bytes(1, &sys.lig, n, 7 + ligand->T, params->topk, nullptr) > 200 * 1024) return DOCK_EINVAL;
    unsigned char *scratch = nullptr;
    const int rc = topk_fixed_scratch(&scratch);
    if (rc != DOCK_OK) return rc;
    cudaStream_t stream = (cudaStream_t)stream_;
    // Nothing in the scratch has to start at zero: both regions the kernel reads are overwritten in full here, in stream
    // order, so whatever the previous call (any ligand) left behind is never seen.
    DOCK_CUDA_CHECK(cudaMemcpyAsync(scratch, blob.bytes.data(), blob.bytes.size(), cudaMemcpyHostToDevice, stream));
    sys.lig = dock_relocate_ligand(blob, scratch);
    DevSystem *sys_dev = (DevSystem *)(scratch + blob.bytes.size());
    DOCK_CUDA_CHECK(cudaMemcpyAsync(sys_dev, &sys, sizeof(sys), cudaMemcpyHostToDevice, stream));
    return launch_topk(sys_dev, 1, &sys.lig, n, 7 + ligand->T, params->topk, params->cluster_rmsd, poses_dev, e_dev,
                       out_idx_dev, out_count_dev, nullptr, nullptr, stream);
}
