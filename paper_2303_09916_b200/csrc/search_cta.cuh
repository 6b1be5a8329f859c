// search_cta.cuh -- the local optimizer of search.cu with a SPECULATIVE LINE SEARCH: one CTA of 4 warps per copy, the four
// warps evaluate four consecutive backtracking trials (alpha, alpha/2, alpha/4, alpha/8) of the same iteration at once.
//
// Why: the paper's own setting is 384 copies x 40 steps; with one warp per copy that is 384 warps on
// 592 schedulers, each running one long dependent chain (profiles/r1l.md: 5.6 % occupancy, 40 ms), and the paper itself
// names the line search as the part of BFGS that "is very time-consuming and cannot be effectively paralleled".
// It can be, across trials: an iteration spends 1.90 evaluations on average, but only 1.10 ROUNDS of four (measured on
// configs[2], profiles/r2c.md), so the sequential evaluations per iteration drop by 1.7x while the otherwise idle SMs do
// the extra, mostly discarded, work.  Every evaluation is the warp evaluator of eval_warp.cuh and warp 0 carries out the
// optimizer's vector arithmetic exactly as local_opt_warp does, so the results are BIT-IDENTICAL to the warp-per-copy
// kernel (tests/test_gpu_parity.py::test_search_kernels_agree_bitwise); only evaluations the sequential algorithm would
// have made are counted.  Barzilai-Borwein has no line search: there the four warps SHARE each evaluation (eval_cta.cuh:
// atoms over the 128 threads, pair rounds over the warps), which changes the order of the force sums -- BB results of
// the two kernels agree to round-off, not bit for bit.
//
// Selected by dock_params.search_kernel (0 = auto: this kernel when n_systems x copies is small, see search.cu).
// (included by search.cu inside its anonymous namespace, after local_opt_warp's helpers)
#pragma once

#include "eval_cta.cuh"

constexpr int CTA_WARPS = 4;
constexpr int CTA_THREADS = CTA_WARPS * 32;

struct SpecBuf {
    float *x, *g, *d, *y, *hy, *H;      // the optimizer's state, written by warp 0 only
    float *xt, *gt, *scratch;           // per warp: trial pose, its gradient, the evaluator's scratch
    float *f;                           // [W] trial energies
    double *ctl;                        // {g.d, alpha0, stop reason} published by warp 0 at the start of an iteration
    int xt_stride, gt_stride, sc_stride;
};

// floats of shared memory of one copy (excluding cur / best of the MC loop)
__host__ __device__ inline int spec_floats(int T, int n_pad)
{
    const int n = 6 + T, np_ = 7 + T;
    const int eval_sc = 8 * n_pad + 2 * pad4(T) + 40 * T;
    return pad4(np_) + 4 * pad4(n) + pad4(n * n) + CTA_WARPS * (pad4(np_) + pad4(n) + eval_sc) + 8 + 8;
}

__device__ __forceinline__ SpecBuf spec_carve(float *base, int T, int n_pad)
{
    const int n = 6 + T, np_ = 7 + T;
    SpecBuf b;
    b.ctl = reinterpret_cast<double *>(base);  base += 8;        // 4 doubles, 8-byte aligned (base is 16-byte aligned)
    b.f = base;               base += 8;
    b.x = base;               base += pad4(np_);
    b.g = base;               base += pad4(n);
    b.d = base;               base += pad4(n);
    b.y = base;               base += pad4(n);
    b.hy = base;              base += pad4(n);
    b.H = base;               base += pad4(n * n);
    b.xt_stride = pad4(np_);  b.gt_stride = pad4(n);  b.sc_stride = 8 * n_pad + 2 * pad4(T) + 40 * T;
    b.xt = base;              base += CTA_WARPS * b.xt_stride;
    b.gt = base;              base += CTA_WARPS * b.gt_stride;
    b.scratch = base;
    return b;
}

// O8 / O8' as local_opt_warp (same arithmetic, same order, same trace records), line-search trials evaluated four at a time.
template <bool EQ4, bool VEC4, bool TRACE>
__device__ __forceinline__ float local_opt_spec(const DevParams &P, const DevGrid &G, const DevLigand &L,
                                                const SpecBuf &b, int cap, int &iters, int &evals, int &why,
                                                float *itrace = nullptr, int itrace_cap = 0)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int T = L.T, n = 6 + T, np_ = 7 + T;
    const int istride = DOCK_ITER_HEADER + np_ + n + n * n;
    float *const xt_mine = b.xt + warp * b.xt_stride, *const gt_mine = b.gt + warp * b.gt_stride;
    float *const sc_mine = b.scratch + warp * b.sc_stride;
    why = DOCK_EXIT_CAP;
    if (threadIdx.x == 0) {
        const float w = b.x[3], x = b.x[4], y = b.x[5], z = b.x[6];
        const float n2 = w * w + x * x + y * y + z * z;
        if (n2 > 0.f) { const float inv = 1.0f / sqrtf(n2); b.x[3] = w * inv; b.x[4] = x * inv; b.x[5] = y * inv; b.x[6] = z * inv; }
        else { b.x[3] = 1.f; b.x[4] = b.x[5] = b.x[6] = 0.f; }
    }
    __syncthreads();
    float f = 0.0f, alpha = 1.0f, f_best = 0.0f;
    double gp = 0.0;
    bool init = true, fresh = true;
    const bool bb = P.optimizer == 1;
    float *const x_best = b.H;
    int it = 0, trial = 0;
    evals = 0;
    for (;;) {
        // ---- evaluate: the start pose / the BB trial by every warp alike, a line-search round by the four warps ----
        int slot = warp;
        float ft;
        if (init || bb) {
            if (init) for (int k = lane; k < np_; k += 32) xt_mine[k] = b.x[k];
            else pose_add_warp(T, b.x, b.d, alpha, xt_mine);
            __syncwarp();
            if (bb)                                // one evaluation shared by the four warps (eval_cta.cuh); gradient -> slot 0
                ft = eval_pose_cta<EQ4, VEC4>(P, G, L, xt_mine, b.gt, b.scratch, b.sc_stride, reinterpret_cast<double *>(b.f));
            else
                ft = eval_pose_warp<true, EQ4, VEC4>(P, G, L, xt_mine, gt_mine, sc_mine, nullptr);
            __syncthreads();                       // every warp has read x and d before warp 0 moves them
        } else {
            slot = trial & (CTA_WARPS - 1);
            if (slot == 0) {                       // trials `trial` .. `trial + 3`: warp w takes alpha shrink^w
                float aw = alpha;
                for (int k = 0; k < warp; ++k) aw *= P.shrink;
                pose_add_warp(T, b.x, b.d, aw, xt_mine);
                const float fw = eval_pose_warp<true, EQ4, VEC4>(P, G, L, xt_mine, gt_mine, sc_mine, nullptr);
                __syncthreads();                   // every warp has read the previous round's energies
                if (lane == 0) b.f[warp] = fw;
                __syncthreads();
            }
            ft = b.f[slot];
        }
        const float *const xt = b.xt + slot * b.xt_stride, *const gt = b.gt + slot * b.gt_stride;
        ++evals;
        if (init) {
            init = false;
            f = ft;
            if (warp == 0) {
                for (int r = lane; r < n; r += 32) b.g[r] = gt[r];
                if (bb) {
                    for (int k = lane; k < np_; k += 32) x_best[k] = b.x[k];
                    __syncwarp();
                } else set_identity(b.H, n, 1.0f);
            }
            if (bb) f_best = f;
        } else if (bb) {
            if (warp == 0) {
                for (int r = lane; r < n; r += 32) {
                    b.d[r] = alpha * b.d[r];
                    b.y[r] = gt[r] - b.g[r];
                    b.g[r] = gt[r];
                }
                for (int k = lane; k < np_; k += 32) b.x[k] = xt[k];
                if (ft < f_best)
                    for (int k = lane; k < np_; k += 32) x_best[k] = xt[k];
                __syncwarp();
            }
            f = ft;
            if (f < f_best) f_best = f;
            if (TRACE && it < itrace_cap && threadIdx.x == 0) itrace[(size_t)it * istride + 5] = ft;
            ++it;
        } else if ((double)ft - (double)f <= (double)P.c1 * (double)alpha * gp) {   // Armijo: accept the step
            bool upd = false;
            if (warp == 0) {
                double ys = 0.0, yy = 0.0, ss = 0.0;
                for (int r = lane; r < n; r += 32) {
                    const float s = alpha * b.d[r], yv = gt[r] - b.g[r];
                    b.d[r] = s;
                    b.y[r] = yv;
                    ys += (double)yv * (double)s; yy += (double)yv * (double)yv; ss += (double)s * (double)s;
                }
                ys = warp_sum_d(ys); yy = warp_sum_d(yy); ss = warp_sum_d(ss);
                for (int k = lane; k < np_; k += 32) b.x[k] = xt[k];
                for (int r = lane; r < n; r += 32) b.g[r] = gt[r];
                __syncwarp();
                upd = ys > (double)P.curv_eps * sqrt(ss) * sqrt(yy);
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
                    rec[4] = alpha; rec[5] = ft; rec[7] = (float)(trial + 1); rec[8] = upd ? 1.f : 0.f; rec[11] = fresh ? 1.f : 0.f;
                }
            }
            f = ft;
            ++it;
        } else {                                   // backtrack
            if (++trial >= P.max_trials) {         // no acceptable trial: stop
                why = DOCK_EXIT_LINESEARCH;
                if (TRACE && it < itrace_cap && threadIdx.x == 0) {
                    float *rec = itrace + (size_t)it * istride;
                    rec[4] = alpha; rec[5] = ft; rec[6] = (float)DOCK_EXIT_LINESEARCH; rec[7] = (float)trial;
                }
                break;
            }
            alpha *= P.shrink;
            continue;                              // the next trial of this round is already evaluated (or a new round starts)
        }
        // ---- start iteration `it`: warp 0 decides and publishes {stop reason, g.d, alpha0} ----
        if (warp == 0) {
            int stop = 0;
            double gpn = 0.0;
            float a0 = 1.0f;
            if (it >= cap) stop = DOCK_EXIT_CAP;
            else {
                double acc = 0.0;
                for (int r = lane; r < n; r += 32) acc += (double)b.g[r] * (double)b.g[r];
                const double gn2 = warp_sum_d(acc);
                if (TRACE && it < itrace_cap) {     // the state this iteration starts from
                    float *rec = itrace + (size_t)it * istride;
                    if (lane == 0) {
                        rec[0] = f; rec[1] = (float)sqrt(gn2); rec[2] = rec[3] = rec[4] = rec[5] = 0.f;
                        rec[6] = 0.f; rec[7] = 0.f; rec[8] = 0.f; rec[9] = 0.f; rec[10] = fresh ? 1.f : 0.f; rec[11] = fresh ? 1.f : 0.f;
                    }
                    for (int k = lane; k < np_; k += 32) rec[DOCK_ITER_HEADER + k] = b.x[k];
                    for (int k = lane; k < n; k += 32) rec[DOCK_ITER_HEADER + np_ + k] = b.g[k];
                    if (bb)
                        for (int k = lane; k < n; k += 32) {
                            rec[DOCK_ITER_HEADER + np_ + n + k] = it > 0 ? b.d[k] : 0.f;
                            rec[DOCK_ITER_HEADER + np_ + 2 * n + k] = it > 0 ? b.y[k] : 0.f;
                        }
                    else
                        for (int k = lane; k < n * n; k += 32) rec[DOCK_ITER_HEADER + np_ + n + k] = b.H[k];
                }
                if (sqrt(gn2) < (double)P.gtol) {
                    stop = DOCK_EXIT_GTOL;
                    if (TRACE && it < itrace_cap && lane == 0) itrace[(size_t)it * istride + 6] = (float)DOCK_EXIT_GTOL;
                } else if (bb) {
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
                    a0 = (float)al;
                    if (TRACE && it < itrace_cap && lane == 0) {
                        float *rec = itrace + (size_t)it * istride;
                        rec[4] = a0; rec[7] = (float)branch; rec[9] = capped ? 1.f : 0.f;
                    }
                    __syncwarp();
                    for (int r = lane; r < n; r += 32) b.d[r] = -b.g[r];
                    __syncwarp();
                } else {
                    for (int r = lane; r < n; r += 32) {
                        float a = 0.0f;
                        for (int c = 0; c < n; ++c) a = fmaf(b.H[r * n + c], b.g[c], a);
                        b.d[r] = -a;
                    }
                    __syncwarp();
                    acc = 0.0;
                    for (int r = lane; r < n; r += 32) acc += (double)b.g[r] * (double)b.d[r];
                    gpn = warp_sum_d(acc);
                    if (gpn >= 0.0) {               // not a descent direction: reset H = I
                        set_identity(b.H, n, 1.0f);
                        fresh = true;
                        for (int r = lane; r < n; r += 32) b.d[r] = -b.g[r];
                        __syncwarp();
                        gpn = -gn2;
                        if (TRACE && it < itrace_cap && lane == 0) itrace[(size_t)it * istride + 9] = 1.f;
                    }
                    if (fresh) {
                        acc = 0.0;
                        for (int r = lane; r < n; r += 32) acc += (double)b.d[r] * (double)b.d[r];
                        const double dn = sqrt(warp_sum_d(acc));
                        if (dn > 1.0) a0 = (float)(1.0 / dn);
                    }
                    if (TRACE && it < itrace_cap && lane == 0) {
                        float *rec = itrace + (size_t)it * istride;
                        rec[2] = (float)gpn; rec[3] = a0;
                    }
                }
            }
            if (lane == 0) { b.ctl[0] = gpn; b.ctl[1] = (double)a0; b.ctl[2] = (double)stop; }
        }
        __syncthreads();
        const int stop = (int)b.ctl[2];
        if (stop) { if (stop == DOCK_EXIT_GTOL) why = DOCK_EXIT_GTOL; break; }
        gp = b.ctl[0];
        alpha = (float)b.ctl[1];
        trial = 0;
        // (the round that follows begins with a barrier-free read of x and d: they were published by the barrier above;
        // warp 0 overwrites them only after the round's own barrier)
    }
    if (bb) {                                      // non-monotone method: report the best point seen
        __syncthreads();
        if (warp == 0) {
            for (int k = lane; k < np_; k += 32) b.x[k] = x_best[k];
        }
        f = f_best;
    }
    __syncthreads();
    iters = it;
    return f;
}
