// score.cu -- dock_score_batch: fused pose -> coordinates -> interpolated energy + gradient for a
// batch of poses (eq. 2-3 at 198-219).  One THREAD per pose
// (eval_thread.cuh).  The threads never cooperate; the CTA size (1..8 warps) is chosen on the host as
// the one that packs most warps into an SM's shared memory (each CTA also costs 1 KB of reserved smem).
#include <algorithm>
#include <mutex>
#include <vector>

#include "common.cuh"
#include "eval_thread.cuh"
#include "host_compile.cuh"
#include "jit_score.cuh"

namespace {

template <bool WANT_GRAD, bool SCHED_PARAM, bool EQ4>
__global__ void __launch_bounds__(256)
score_thread_kernel(const DevParams P, const DevGrid G, const __grid_constant__ TppLigand L, long long n_poses,
                    const float *__restrict__ poses, float *__restrict__ energy,
                    float *__restrict__ grad, float *__restrict__ terms, int warp_floats)
{
    extern __shared__ float smem_all[];
    float *const smem = smem_all + (size_t)(threadIdx.x >> 5) * warp_floats;
    const int np_ = 7 + L.T, ng = 6 + L.T;
    // idle lanes of the last warp redo the last pose: same inputs, same bits, same stores (benign)
    const long long p = min((long long)blockIdx.x * blockDim.x + threadIdx.x, n_poses - 1);
    EvalTerms t;
    const float e = eval_pose_thread<WANT_GRAD, SCHED_PARAM, EQ4>(P, G, L, poses + p * np_, 1, grad + p * ng, 1, smem, t);
    energy[p] = e;
    if (terms) { terms[3 * p] = t.e_grid; terms[3 * p + 1] = t.e_wall; terms[3 * p + 2] = t.e_intra; }
}

struct ScorePlan {
    DevParams P;
    DevGrid G;
    TppLigand L;
    std::vector<uint4> overflow;
    size_t need;
};

int plan_score(const dock_params *params, const dock_grid *grid, const dock_ligand *lig, ScorePlan &pl)
{
    if (dock_make_dev_params(params, &pl.P) != DOCK_OK) return DOCK_EINVAL;
    if (dock_make_dev_grid(params, grid, &pl.G) != DOCK_OK) return DOCK_EINVAL;
    if (dock_compile_tpp(params, grid, lig, pl.L, pl.overflow) != DOCK_OK) return DOCK_EINVAL;
    pl.need = align_up(pl.overflow.size() * sizeof(uint4) + 16, 256);
    return DOCK_OK;
}

template <bool WANT_GRAD, bool SCHED_PARAM, bool EQ4 = false>
int launch(const ScorePlan &pl, long long n_poses, const float *poses_dev, float *energy_dev, float *grad_dev,
           float *terms_dev, cudaStream_t stream)
{
    auto kern = score_thread_kernel<WANT_GRAD, SCHED_PARAM, EQ4>;
    const int warp_floats = tpp_warp_floats(pl.L.N, pl.L.T, WANT_GRAD, pl.L.fm_alias != 0);
    const size_t warp_bytes = (size_t)warp_floats * sizeof(float);
    if (warp_bytes > 227 * 1024) return DOCK_EINVAL;
    // CTA size: most resident warps per SM (shared memory + 1 KB reserved per CTA, registers), ties -> fewer warps per CTA
    if (warp_bytes > 48 * 1024 / 8)
        DOCK_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)std::min<size_t>(8 * warp_bytes, 227 * 1024)));
    int best_w = 1, best_res = 0;
    for (int w = 1; w <= 8; ++w) {
        if (w * warp_bytes > 227 * 1024) break;
        int ctas = 0;
        DOCK_CUDA_CHECK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&ctas, kern, 32 * w, w * warp_bytes));
        if (ctas * w > best_res) { best_res = ctas * w; best_w = w; }
    }
    if (best_res == 0) return DOCK_EINVAL;
    const size_t smem = best_w * warp_bytes;
    const long long per_cta = 32LL * best_w;
    const long long blocks = (n_poses + per_cta - 1) / per_cta;
    if (blocks > 0x7fffffffLL) return DOCK_EINVAL;
    kern<<<(unsigned)blocks, (unsigned)per_cta, smem, stream>>>(pl.P, pl.G, pl.L, n_poses, poses_dev, energy_dev, grad_dev, terms_dev, warp_floats);
    DOCK_LAUNCH_CHECK();
    return DOCK_OK;
}

// `ws` receives the overflow schedule (if any); pl.L.sched_global is pointed at it.
int score_launch(ScorePlan &pl, long long n_poses, const float *poses_dev, float *energy_dev, float *grad_dev,
                 float *terms_dev, void *ws, cudaStream_t stream, bool upload = true)
{
    if (n_poses < 1) return DOCK_OK;
    if (!pl.L.sched_in_param) {
        if (upload)
            DOCK_CUDA_CHECK(cudaMemcpyAsync(ws, pl.overflow.data(), pl.overflow.size() * sizeof(uint4),
                                            cudaMemcpyHostToDevice, stream));
        pl.L.sched_global = (const uint4 *)ws;
        if (grad_dev && pl.G.channels == 4) return launch<true, false, true>(pl, n_poses, poses_dev, energy_dev, grad_dev, terms_dev, stream);
        return grad_dev ? launch<true, false>(pl, n_poses, poses_dev, energy_dev, grad_dev, terms_dev, stream)
                        : launch<false, false>(pl, n_poses, poses_dev, energy_dev, grad_dev, terms_dev, stream);
    }
    if (grad_dev && pl.G.channels == 4) return launch<true, true, true>(pl, n_poses, poses_dev, energy_dev, grad_dev, terms_dev, stream);
    return grad_dev ? launch<true, true>(pl, n_poses, poses_dev, energy_dev, grad_dev, terms_dev, stream)
                    : launch<false, true>(pl, n_poses, poses_dev, energy_dev, grad_dev, terms_dev, stream);
}

// Copy streams and events of dock_score_batch_host: the only resources the library owns.  One context per device,
// created on first use under a mutex and published only when every create call has succeeded; the pipeline itself runs
// under the context's mutex, so concurrent host threads serialise per device.
constexpr int MAX_CHUNKS = 8;
constexpr int MAX_DEVICES = 64;
struct HostPipe {
    std::mutex mu;
    bool ready = false;
    cudaStream_t s_in = nullptr, s_out = nullptr;
    cudaEvent_t ev_in[MAX_CHUNKS], ev_k[MAX_CHUNKS], ev_begin, ev_end;
};
HostPipe g_pipes[MAX_DEVICES];

int pipe_init(HostPipe &hp)
{
    if (hp.ready) return DOCK_OK;
    cudaStream_t a = nullptr, b = nullptr;
    cudaEvent_t ev[2 * MAX_CHUNKS + 2];
    int made = 0;
    cudaError_t e = cudaStreamCreateWithFlags(&a, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&b, cudaStreamNonBlocking);
    for (; e == cudaSuccess && made < 2 * MAX_CHUNKS + 2; ++made) e = cudaEventCreateWithFlags(&ev[made], cudaEventDisableTiming);
    if (e != cudaSuccess) {                                  // roll back: nothing half-initialised is ever published
        for (int k = 0; k < made - 1; ++k) cudaEventDestroy(ev[k]);
        if (a) cudaStreamDestroy(a);
        if (b) cudaStreamDestroy(b);
        g_dock_last_cuda_error.store((int)e);
        return DOCK_ECUDA;
    }
    hp.s_in = a; hp.s_out = b;
    for (int c = 0; c < MAX_CHUNKS; ++c) { hp.ev_in[c] = ev[2 * c]; hp.ev_k[c] = ev[2 * c + 1]; }
    hp.ev_begin = ev[2 * MAX_CHUNKS]; hp.ev_end = ev[2 * MAX_CHUNKS + 1];
    hp.ready = true;
    return DOCK_OK;
}

// The ligand-specialised kernel (jit_score.cu) is opt-in: it costs a run-time compilation per ligand (0.4-6 s, cached) and
// gains 1.15x on BASELINE configs[1] (profiles/r2b.md), so score_kernel = 0 keeps the generic kernel.
bool use_jit(const dock_params *params, const dock_grid *grid, const dock_ligand *lig, int64_t n_poses)
{
    return params->score_kernel == 2 && n_poses >= 1 && lig && grid;
}

}  // namespace

extern "C" int dock_score_batch(const dock_params *params, const dock_grid *grid, const dock_ligand *ligand,
                                int64_t n_poses, const float *poses_dev,
                                float *energy_dev, float *grad_dev, float *terms_dev,
                                void *ws_dev, size_t ws_bytes, size_t *needed, void *stream_)
{
    ScorePlan pl;
    const int rc = plan_score(params, grid, ligand, pl);
    if (rc != DOCK_OK) return rc;
    if (n_poses < 0) return DOCK_EINVAL;
    if (needed) *needed = pl.need;
    if (!ws_dev || ws_bytes < pl.need) return DOCK_EWORKSPACE;
    if (n_poses > 0 && (!poses_dev || !energy_dev)) return DOCK_EINVAL;
    if (use_jit(params, grid, ligand, n_poses)) {
        const int rj = jit_score_launch(params, grid, ligand, pl.P, pl.G, n_poses, poses_dev, energy_dev, grad_dev, terms_dev,
                                        (cudaStream_t)stream_);
        if (rj == DOCK_OK || params->score_kernel == 2) return rj;      // forced: report the failure; auto: generic kernel
    }
    return score_launch(pl, n_poses, poses_dev, energy_dev, grad_dev, terms_dev, ws_dev, (cudaStream_t)stream_);
}

extern "C" int dock_score_batch_host(const dock_params *params, const dock_grid *grid, const dock_ligand *ligand,
                                     int64_t n_poses, const float *poses_host,
                                     float *energy_host, float *grad_host, float *terms_host,
                                     void *ws_dev, size_t ws_bytes, size_t *needed, void *stream_)
{
    ScorePlan pl;
    const int rc = plan_score(params, grid, ligand, pl);
    if (rc != DOCK_OK) return rc;
    if (n_poses < 0) return DOCK_EINVAL;
    const int np_ = 7 + ligand->T, ng = 6 + ligand->T;
    const size_t b_blob = pl.need;
    const size_t b_pose = align_up((size_t)n_poses * np_ * sizeof(float), 256);
    const size_t b_e = align_up((size_t)n_poses * sizeof(float), 256);
    const size_t b_g = grad_host ? align_up((size_t)n_poses * ng * sizeof(float), 256) : 0;
    const size_t b_t = terms_host ? align_up((size_t)n_poses * 3 * sizeof(float), 256) : 0;
    const size_t need = b_blob + b_pose + b_e + b_g + b_t;
    if (needed) *needed = need;
    if (!ws_dev || ws_bytes < need) return DOCK_EWORKSPACE;
    if (n_poses > 0 && (!poses_host || !energy_host)) return DOCK_EINVAL;
    if (n_poses == 0) return DOCK_OK;
    cudaStream_t stream = (cudaStream_t)stream_;
    unsigned char *ws = (unsigned char *)ws_dev;
    float *d_pose = (float *)(ws + b_blob), *d_e = (float *)(ws + b_blob + b_pose);
    float *d_g = grad_host ? (float *)(ws + b_blob + b_pose + b_e) : nullptr;
    float *d_t = terms_host ? (float *)(ws + b_blob + b_pose + b_e + b_g) : nullptr;
    // Three-stage pipeline over chunks of the batch: host->device copies on one side stream, kernels on the
    // caller's stream, device->host copies on another side stream, so that PCIe in, compute and PCIe out
    // overlap (the buses are full duplex).  The side streams and events belong to the library (one set per device).
    int dev = 0;
    DOCK_CUDA_CHECK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= MAX_DEVICES) return DOCK_EINVAL;
    HostPipe &hp = g_pipes[dev];
    std::lock_guard<std::mutex> lock(hp.mu);
    if (pipe_init(hp) != DOCK_OK) return DOCK_ECUDA;
    const int n_chunks = (int)std::min<int64_t>(MAX_CHUNKS, (n_poses + 65535) / 65536);      // >= 64 Ki poses per chunk
    const int64_t per = ((n_poses + n_chunks - 1) / n_chunks + 31) / 32 * 32;
    // on any failure the copies already enqueued are drained before returning: the caller's host buffers must not be
    // written after the call has come back
    const bool jit = use_jit(params, grid, ligand, n_poses);
    bool uploaded = false;
    auto pipeline = [&]() -> int {
        DOCK_CUDA_CHECK(cudaEventRecord(hp.ev_begin, stream));              // the workspace may still be in use upstream
        DOCK_CUDA_CHECK(cudaStreamWaitEvent(hp.s_in, hp.ev_begin, 0));
        DOCK_CUDA_CHECK(cudaStreamWaitEvent(hp.s_out, hp.ev_begin, 0));
        for (int c = 0; c < n_chunks; ++c) {
            const int64_t o = c * per, m = std::min<int64_t>(per, n_poses - o);
            if (m <= 0) break;
            DOCK_CUDA_CHECK(cudaMemcpyAsync(d_pose + o * np_, poses_host + o * np_, (size_t)m * np_ * sizeof(float), cudaMemcpyHostToDevice, hp.s_in));
            DOCK_CUDA_CHECK(cudaEventRecord(hp.ev_in[c], hp.s_in));
            DOCK_CUDA_CHECK(cudaStreamWaitEvent(stream, hp.ev_in[c], 0));
            int rc2 = DOCK_EINVAL;
            if (jit) rc2 = jit_score_launch(params, grid, ligand, pl.P, pl.G, m, d_pose + o * np_, d_e + o, d_g ? d_g + o * ng : nullptr,
                                            d_t ? d_t + o * 3 : nullptr, stream);
            if (rc2 != DOCK_OK && !(jit && params->score_kernel == 2))
                rc2 = score_launch(pl, m, d_pose + o * np_, d_e + o, d_g ? d_g + o * ng : nullptr, d_t ? d_t + o * 3 : nullptr,
                                   ws, stream, !uploaded), uploaded = true;
            if (rc2 != DOCK_OK) return rc2;
            DOCK_CUDA_CHECK(cudaEventRecord(hp.ev_k[c], stream));
            DOCK_CUDA_CHECK(cudaStreamWaitEvent(hp.s_out, hp.ev_k[c], 0));
            DOCK_CUDA_CHECK(cudaMemcpyAsync(energy_host + o, d_e + o, (size_t)m * sizeof(float), cudaMemcpyDeviceToHost, hp.s_out));
            if (grad_host) DOCK_CUDA_CHECK(cudaMemcpyAsync(grad_host + o * ng, d_g + o * ng, (size_t)m * ng * sizeof(float), cudaMemcpyDeviceToHost, hp.s_out));
            if (terms_host) DOCK_CUDA_CHECK(cudaMemcpyAsync(terms_host + o * 3, d_t + o * 3, (size_t)m * 3 * sizeof(float), cudaMemcpyDeviceToHost, hp.s_out));
        }
        DOCK_CUDA_CHECK(cudaEventRecord(hp.ev_end, hp.s_out));
        DOCK_CUDA_CHECK(cudaStreamWaitEvent(stream, hp.ev_end, 0));
        return DOCK_OK;
    };
    const int rc3 = pipeline();
    if (rc3 != DOCK_OK) {
        cudaStreamSynchronize(hp.s_in);
        cudaStreamSynchronize(stream);
        cudaStreamSynchronize(hp.s_out);
        return rc3;
    }
    DOCK_CUDA_CHECK(cudaStreamSynchronize(stream));
    return DOCK_OK;
}
