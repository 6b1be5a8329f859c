// score.cu -- dock_score_batch: fused pose -> coordinates -> interpolated energy + gradient for a
// batch of poses (eq. 2-3 at 198-219).  One warp per pose.
#include <vector>

#include "common.cuh"
#include "eval.cuh"
#include "host_compile.cuh"

namespace {

constexpr int SCORE_WARPS = 8;

template <bool WANT_GRAD>
__global__ void __launch_bounds__(SCORE_WARPS * 32)
score_warp_kernel(DevParams P, DevGrid G, DevLigand L, long long n_poses, int warp_floats,
                  const float *__restrict__ poses, float *__restrict__ energy,
                  float *__restrict__ grad, float *__restrict__ terms)
{
    extern __shared__ float smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int np_ = 7 + L.T, ng = 6 + L.T;
    float *pose_s = smem + (size_t)warp * warp_floats;
    float *grad_s = pose_s + ((np_ + 3) & ~3);
    float *scratch = grad_s + ((ng + 3) & ~3);
    const long long stride = (long long)gridDim.x * SCORE_WARPS;
    for (long long p = (long long)blockIdx.x * SCORE_WARPS + warp; p < n_poses; p += stride) {
        for (int k = lane; k < np_; k += 32) pose_s[k] = __ldg(&poses[p * np_ + k]);
        __syncwarp();
        EvalTerms t;
        const float e = eval_pose_warp<WANT_GRAD>(P, G, L, pose_s, grad_s, scratch, &t);
        if (lane == 0) {
            energy[p] = e;
            if (terms) { terms[3 * p] = t.e_grid; terms[3 * p + 1] = t.e_wall; terms[3 * p + 2] = t.e_intra; }
        }
        if (WANT_GRAD)
            for (int k = lane; k < ng; k += 32) grad[p * ng + k] = grad_s[k];
        __syncwarp();
    }
}

struct ScorePlan {
    DevParams P;
    DevGrid G;
    LigandBlob blob;
    size_t need;
};

int plan_score(const dock_params *params, const dock_grid *grid, const dock_ligand *lig, ScorePlan &pl)
{
    if (dock_make_dev_params(params, &pl.P) != DOCK_OK) return DOCK_EINVAL;
    if (dock_make_dev_grid(grid, &pl.G) != DOCK_OK) return DOCK_EINVAL;
    if (dock_compile_ligand(params, grid, lig, pl.blob) != DOCK_OK) return DOCK_EINVAL;
    pl.need = pl.blob.bytes.size();
    return DOCK_OK;
}

}  // namespace

int dock_score_launch(const DevParams &P, const DevGrid &G, const DevLigand &L, long long n_poses,
                      const float *poses_dev, float *energy_dev, float *grad_dev, float *terms_dev,
                      cudaStream_t stream)
{
    const int np_ = 7 + L.T, ng = 6 + L.T;
    const int warp_floats = ((np_ + 3) & ~3) + ((ng + 3) & ~3) + eval_scratch_floats(L.n_pad, L.T);
    const size_t smem = (size_t)SCORE_WARPS * warp_floats * sizeof(float);
    long long blocks = (n_poses + SCORE_WARPS - 1) / SCORE_WARPS;
    const long long max_blocks = 148LL * 8 * 16;   // grid-stride beyond this
    if (blocks > max_blocks) blocks = max_blocks;
    if (blocks < 1) return DOCK_OK;
    if (grad_dev) {
        if (smem > 48 * 1024)
            DOCK_CUDA_CHECK(cudaFuncSetAttribute(score_warp_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        score_warp_kernel<true><<<(unsigned)blocks, SCORE_WARPS * 32, smem, stream>>>(P, G, L, n_poses, warp_floats, poses_dev, energy_dev, grad_dev, terms_dev);
    } else {
        if (smem > 48 * 1024)
            DOCK_CUDA_CHECK(cudaFuncSetAttribute(score_warp_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        score_warp_kernel<false><<<(unsigned)blocks, SCORE_WARPS * 32, smem, stream>>>(P, G, L, n_poses, warp_floats, poses_dev, energy_dev, grad_dev, terms_dev);
    }
    DOCK_LAUNCH_CHECK();
    return DOCK_OK;
}

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
    cudaStream_t stream = (cudaStream_t)stream_;
    DOCK_CUDA_CHECK(cudaMemcpyAsync(ws_dev, pl.blob.bytes.data(), pl.blob.bytes.size(), cudaMemcpyHostToDevice, stream));
    const DevLigand L = dock_relocate_ligand(pl.blob, (const unsigned char *)ws_dev);
    return dock_score_launch(pl.P, pl.G, L, n_poses, poses_dev, energy_dev, grad_dev, terms_dev, stream);
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
    const size_t b_blob = align_up(pl.need, 256);
    const size_t b_pose = align_up((size_t)n_poses * np_ * sizeof(float), 256);
    const size_t b_e = align_up((size_t)n_poses * sizeof(float), 256);
    const size_t b_g = grad_host ? align_up((size_t)n_poses * ng * sizeof(float), 256) : 0;
    const size_t b_t = terms_host ? align_up((size_t)n_poses * 3 * sizeof(float), 256) : 0;
    const size_t need = b_blob + b_pose + b_e + b_g + b_t;
    if (needed) *needed = need;
    if (!ws_dev || ws_bytes < need) return DOCK_EWORKSPACE;
    if (n_poses > 0 && (!poses_host || !energy_host)) return DOCK_EINVAL;
    cudaStream_t stream = (cudaStream_t)stream_;
    unsigned char *ws = (unsigned char *)ws_dev;
    float *d_pose = (float *)(ws + b_blob), *d_e = (float *)(ws + b_blob + b_pose);
    float *d_g = grad_host ? (float *)(ws + b_blob + b_pose + b_e) : nullptr;
    float *d_t = terms_host ? (float *)(ws + b_blob + b_pose + b_e + b_g) : nullptr;
    DOCK_CUDA_CHECK(cudaMemcpyAsync(ws, pl.blob.bytes.data(), pl.blob.bytes.size(), cudaMemcpyHostToDevice, stream));
    DOCK_CUDA_CHECK(cudaMemcpyAsync(d_pose, poses_host, (size_t)n_poses * np_ * sizeof(float), cudaMemcpyHostToDevice, stream));
    const DevLigand L = dock_relocate_ligand(pl.blob, ws);
    const int rc2 = dock_score_launch(pl.P, pl.G, L, n_poses, d_pose, d_e, d_g, d_t, stream);
    if (rc2 != DOCK_OK) return rc2;
    DOCK_CUDA_CHECK(cudaMemcpyAsync(energy_host, d_e, (size_t)n_poses * sizeof(float), cudaMemcpyDeviceToHost, stream));
    if (grad_host) DOCK_CUDA_CHECK(cudaMemcpyAsync(grad_host, d_g, (size_t)n_poses * ng * sizeof(float), cudaMemcpyDeviceToHost, stream));
    if (terms_host) DOCK_CUDA_CHECK(cudaMemcpyAsync(terms_host, d_t, (size_t)n_poses * 3 * sizeof(float), cudaMemcpyDeviceToHost, stream));
    DOCK_CUDA_CHECK(cudaStreamSynchronize(stream));
    return DOCK_OK;
}
