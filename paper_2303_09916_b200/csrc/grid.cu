// grid.cu -- A1: per-type grid maps over protein atoms binned into cells (eq. 2's inner
// sum at PAPER.md:198-199).
//
//   G[m][iz][iy][ix] = sum_{j : |node - r_j| < cutoff} f(lig_types[m], type_j, |node - r_j|)
//
// Host: protein atoms are binned into cubic cells of edge = cutoff + 0.01 A over the box grown by the cutoff
// (counting sort, stable -> fixed summation order).  Device: one thread per node, a warp covers a
// compact 4x4x2 block of nodes so that its lanes share almost the same in-range atom set: the warp collects
// the atoms near its block once (shared-memory candidate list), then each thread walks the list, decides
// r < cutoff (fp32, redone in double within round-off of the cutoff: DESIGN.md D-CUT) and accumulates up to 8 maps in registers.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <vector>

#include "common.cuh"
#include "host_compile.cuh"

namespace {

constexpr int MAPS_PER_PASS = 8;

// Per-system part of the arguments; an array of these lives in the workspace so that ONE launch covers all systems
// of a screening batch (BASELINE.json configs[3]).
struct GridSysArgs {
    int   nx, ny, nz;
    float ox, oy, oz, h;
    float clo[3];          // low corner of the cell lattice
    float inv_cell;        // 1 / cell edge
    int   ncx, ncy, ncz;
    int   atoms_off;       // first atom of this system in GridBuildArgs::atoms
    int   cells_off;       // first cell of this system in GridBuildArgs::cell_start (entries are system-local atom indices)
    int   block_begin;     // first value of blockIdx.x that belongs to this system
    int   pad_;
    float *out;            // [n_maps][channels][nz][ny][nx]
    Cell8 *packed;         // gather image of the same maps
    float4 *quad;          // 4-corner image (single-channel maps), or NULL
};

struct GridBuildArgs {
    float cutoff, cutoff2;
    int   n_maps, n_types;
    float w[5];
    const float4 *atoms;   // all systems, each sorted by cell; w = bitcast(type)
    const int    *cell_start;
    const float4 *pair_tab;// [n_maps][n_types] {rsum, wh, whb, 0}
    int   channels;        // 1, or 4 = (score, d/dx, d/dy, d/dz): eq. 4's per-vertex gradients (NEXT-2)
    // maps are processed in order of ligand radius: slot k writes map map_of[k]; bit k of fresh says that slot k
    // has another radius than slot k-1 (or opens a pass), i.e. the distance-only part of the term must be recomputed.
    // The two Gaussians and the repulsion depend on the ligand type only through its radius.
    int      map_of[DOCK_MAX_XS_TYPES];
    unsigned fresh;
    const GridSysArgs *sys;
    int   n_sys;
};

// r < cutoff for node (ix,iy,iz) at origin + h i and an atom, every operation in double with products and sums rounded
// separately (no contraction).  Rare path of grid_build_kernel: kept out of line so that it costs the hot loop no registers.
__device__ __noinline__ bool in_range_exact(float ox, float oy, float oz, float h, int ix, int iy, int iz,
                                            float ax, float ay, float az, float cutoff)
{
    const double ddx = __dsub_rn(__dadd_rn((double)ox, __dmul_rn((double)h, (double)ix)), (double)ax);
    const double ddy = __dsub_rn(__dadd_rn((double)oy, __dmul_rn((double)h, (double)iy)), (double)ay);
    const double ddz = __dsub_rn(__dadd_rn((double)oz, __dmul_rn((double)h, (double)iz)), (double)az);
    const double rr = __dsqrt_rn(__dadd_rn(__dadd_rn(__dmul_rn(ddx, ddx), __dmul_rn(ddy, ddy)), __dmul_rn(ddz, ddz)));
    return rr < (double)cutoff;
}

constexpr int GRID_CAND = 256;       // candidate atoms a warp collects before it evaluates them

// One warp owns a 4 x 4 x 2 block of nodes.  Its lanes first scan the cells around the block TOGETHER -- lane l
// tests atom j0 + l against the block's centre with the cutoff grown by the block's half-diagonal -- and compact the
// survivors, in atom order, into a shared-memory list; then every lane walks that list for its own node.  A node's
// own 27 cells hold about 6.5 times as many atoms as its cutoff sphere, the list about 1.3 times (profiles/r1k.md).
template <bool GRAD>
__global__ void __launch_bounds__(128) grid_build_kernel(GridBuildArgs A)
{
    __shared__ float4 tab[MAPS_PER_PASS * DOCK_MAX_XS_TYPES];
    __shared__ float4 cand_all[4][GRID_CAND];
    __shared__ GridSysArgs S;
    const int m0 = blockIdx.y * MAPS_PER_PASS;
    const int nm = min(MAPS_PER_PASS, A.n_maps - m0);
    for (int k = threadIdx.x; k < nm * A.n_types; k += blockDim.x) tab[k] = A.pair_tab[m0 * A.n_types + k];
    if (threadIdx.x == 0) {                                           // the system this block belongs to
        int lo = 0, hi = A.n_sys - 1;
        while (lo < hi) {
            const int mid = (lo + hi + 1) >> 1;
            if ((int)blockIdx.x >= __ldg(&A.sys[mid].block_begin)) lo = mid; else hi = mid - 1;
        }
        S = A.sys[lo];
    }
    __syncthreads();

    // block tile 8 x 8 x 2 nodes; warp tile 4 x 4 x 2
    const int tbx = (S.nx + 7) / 8, tby = (S.ny + 7) / 8;
    const int bl = (int)blockIdx.x - S.block_begin;
    const int bx = bl % tbx, by = (bl / tbx) % tby, bz = bl / (tbx * tby);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int wx0 = bx * 8 + (warp & 1) * 4, wy0 = by * 8 + (warp >> 1) * 4, wz0 = bz * 2;
    if (wx0 >= S.nx || wy0 >= S.ny || wz0 >= S.nz) return;            // whole warp outside the lattice
    const int ix = wx0 + (lane & 3), iy = wy0 + ((lane >> 2) & 3), iz = wz0 + (lane >> 4);
    const bool live = ix < S.nx && iy < S.ny && iz < S.nz;
    float4 *cand = cand_all[warp];
    const float4 *atoms = A.atoms + S.atoms_off;
    const int *cell_start = A.cell_start + S.cells_off;

    // node coordinate in fp32: fmaf(i, h, origin); r^2 < cutoff^2 is decided on it unless it is within round-off of the
    // threshold, where the decision is redone in double (flush(), DESIGN.md D-CUT)
    const float mx = __fmaf_rn((float)ix, S.h, S.ox);
    const float my = __fmaf_rn((float)iy, S.h, S.oy);
    const float mz = __fmaf_rn((float)iz, S.h, S.oz);
    // the warp's block: centre, and the cutoff grown by its half-diagonal (1.5, 1.5, 0.5 spacings) plus a guard band
    const float cxw = fmaf((float)wx0 + 1.5f, S.h, S.ox), cyw = fmaf((float)wy0 + 1.5f, S.h, S.oy), czw = fmaf((float)wz0 + 0.5f, S.h, S.oz);
    const float reach = A.cutoff + 2.18f * S.h + 0.01f;
    const float reach2 = reach * reach;
    const int cx_lo = max((int)floorf((cxw - reach - S.clo[0]) * S.inv_cell), 0), cx_hi = min((int)floorf((cxw + reach - S.clo[0]) * S.inv_cell), S.ncx - 1);
    const int cy_lo = max((int)floorf((cyw - reach - S.clo[1]) * S.inv_cell), 0), cy_hi = min((int)floorf((cyw + reach - S.clo[1]) * S.inv_cell), S.ncy - 1);
    const int cz_lo = max((int)floorf((czw - reach - S.clo[2]) * S.inv_cell), 0), cz_hi = min((int)floorf((czw + reach - S.clo[2]) * S.inv_cell), S.ncz - 1);

    // |r2_fp32 - r2_exact| <= 2 sqrt(3) r (ulp(node coordinate) / 2 + ulp(8) / 2) + 3 ulp(r2) < 14 r_cut/8 2^-23 c_max + 2e-5, c_max the
    // largest |node coordinate| of this lattice: well inside 1e-3 A^2 up to c_max ~ 260 A; beyond, the window grows with c_max
    // (32 x 2^-23 c_max, a factor 2 of margin) so that a box far from the origin keeps the exact decision too
    const float cmax = fmaxf(fmaxf(fmaxf(fabsf(S.ox), fabsf(fmaf((float)(S.nx - 1), S.h, S.ox))),
                                   fmaxf(fabsf(S.oy), fabsf(fmaf((float)(S.ny - 1), S.h, S.oy)))),
                             fmaxf(fabsf(S.oz), fabsf(fmaf((float)(S.nz - 1), S.h, S.oz))));
    const float cut_window = fmaxf(1e-3f, 3.8e-6f * cmax);
    float acc[MAPS_PER_PASS], agx[MAPS_PER_PASS], agy[MAPS_PER_PASS], agz[MAPS_PER_PASS];
#pragma unroll
    for (int m = 0; m < MAPS_PER_PASS; ++m) acc[m] = agx[m] = agy[m] = agz[m] = 0.0f;

    // every lane adds the listed atoms to its own node, in list (= atom) order
    auto flush = [&](int n_cand) {
        __syncwarp();
        if (live)
            for (int k = 0; k < n_cand; ++k) {
                const float4 a = cand[k];
                const float fx = __fsub_rn(mx, a.x), fy = __fsub_rn(my, a.y), fz = __fsub_rn(mz, a.z);
                const float r2 = __fmaf_rn(fz, fz, __fmaf_rn(fy, fy, __fmul_rn(fx, fx)));
                bool in_range = r2 < A.cutoff2;
                if (fabsf(r2 - A.cutoff2) < cut_window) {
                    // Within fp32 round-off of the cutoff sphere (about one node-atom pair in 150): the vertex score jumps by
                    // f(cutoff^-) ~ -0.004 there (reading S3), so the decision is taken as the definition states it -- r < cutoff
                    // with the node at origin + h i and every operation in double, products and sums rounded separately
                    in_range = in_range_exact(S.ox, S.oy, S.oz, S.h, ix, iy, iz, a.x, a.y, a.z, A.cutoff);
                }
                if (in_range) {
                    const float r = sqrtf(r2);
                    const int tj = __float_as_int(a.w);
                    float d = 0.f, dm3 = 0.f, rep = 0.f, base = 0.f, dbase = 0.f;
#pragma unroll
                    for (int m = 0; m < MAPS_PER_PASS; ++m) {
                        if (m < nm) {
                            const float4 t = tab[m * A.n_types + tj];
                            if ((A.fresh >> (m0 + m)) & 1u) {             // uniform: a new ligand radius
                                d = r - t.x;
                                const float g1 = A.w[0] * fast_ex2(-5.770780163555854f * d * d);
                                dm3 = d - 3.0f;
                                const float g2 = A.w[1] * fast_ex2(-0.36067376022224085f * dm3 * dm3);
                                rep = fminf(d, 0.0f);
                                base = fmaf(A.w[2] * rep, rep, g1 + g2);
                                if (GRAD) dbase = fmaf(-8.0f * d, g1, fmaf(-0.5f * dm3, g2, 2.0f * A.w[2] * rep));
                            }
                            float e = fmaf(t.y, __saturatef(1.5f - d), base);
                            e = fmaf(t.z, __saturatef(d * -1.4285714285714286f), e);
                            acc[m] += e;
                            if (GRAD) {                                   // d f / d(vertex) = f'(r) (m - r_j) / r
                                float de = dbase;
                                de -= (d >= 0.5f && d < 1.5f) ? t.y : 0.0f;
                                de -= (d >= -0.7f && d < 0.0f) ? t.z * 1.4285714285714286f : 0.0f;
                                const float k2 = r > 0.0f ? de / r : 0.0f;
                                agx[m] = fmaf(k2, fx, agx[m]); agy[m] = fmaf(k2, fy, agy[m]); agz[m] = fmaf(k2, fz, agz[m]);
                            }
                        }
                    }
                }
            }
        __syncwarp();
    };

    int n_cand = 0;
    for (int zc = cz_lo; zc <= cz_hi; ++zc)
        for (int yc = cy_lo; yc <= cy_hi; ++yc) {
            // the x-cells of a row are contiguous in the sorted atom array
            const int base = (zc * S.ncy + yc) * S.ncx;
            const int j0 = __ldg(&cell_start[base + cx_lo]), j1 = __ldg(&cell_start[base + cx_hi + 1]);
            for (int jb = j0; jb < j1; jb += 32) {
                const int j = jb + lane;
                float4 a = make_float4(0.f, 0.f, 0.f, 0.f);
                bool near = false;
                if (j < j1) {
                    a = __ldg(&atoms[j]);
                    const float dx = a.x - cxw, dy = a.y - cyw, dz = a.z - czw;
                    near = fmaf(dz, dz, fmaf(dy, dy, dx * dx)) < reach2;
                }
                const unsigned mask = __ballot_sync(FULL_MASK, near);
                if (n_cand + __popc(mask) > GRID_CAND) { flush(n_cand); n_cand = 0; }
                if (near) cand[n_cand + __popc(mask & ((1u << lane) - 1u))] = a;
                n_cand += __popc(mask);
            }
        }
    flush(n_cand);
    if (!live) return;

    const size_t nodes = (size_t)S.nx * S.ny * S.nz;
    const size_t node = ((size_t)iz * S.ny + iy) * S.nx + ix;
#pragma unroll
    for (int m = 0; m < MAPS_PER_PASS; ++m)
        if (m < nm) {
            float *o = S.out + (size_t)A.map_of[m0 + m] * A.channels * nodes + node;
            o[0] = acc[m];
            if (GRAD) { o[nodes] = agx[m]; o[2 * nodes] = agy[m]; o[3 * nodes] = agz[m]; }
        }
}

// Gather layout (Cell8, common.cuh): entry (ix,iy,iz) of map m = the 8 corners of the cell whose low corner is that
// node (indices clamped to the last node).  Pure data movement: values are bit-identical copies.
__global__ void __launch_bounds__(256) grid_pack_kernel(const GridSysArgs *__restrict__ sys, int maps_x_channels)
{
    // blockIdx.y = system; one thread per entry; consecutive threads walk x -> coalesced reads, 32-byte stores
    const GridSysArgs S = sys[blockIdx.y];
    const int nx = S.nx, ny = S.ny, nz = S.nz;
    const float *__restrict__ plain = S.out;
    Cell8 *__restrict__ packed = S.packed;
    const long long rows = (long long)maps_x_channels * nz * ny;
    const long long total = rows * nx;
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (long long)gridDim.x * blockDim.x) {
        const int ix = (int)(e % nx);
        const long long row = e / nx;                 // (m * nz + iz) * ny + iy
        const int iy = (int)(row % ny);
        const int iz = (int)((row / ny) % nz);
        const long long up = (iy + 1 < ny) ? nx : 0;
        const long long fw = (iz + 1 < nz) ? (long long)nx * ny : 0;
        const int rt = (ix + 1 < nx) ? 1 : 0;
        const float *q = plain + e;
        Cell8 c;
        c.lo = make_float4(__ldg(q), __ldg(q + rt), __ldg(q + up), __ldg(q + up + rt));
        c.hi = make_float4(__ldg(q + fw), __ldg(q + fw + rt), __ldg(q + fw + up), __ldg(q + fw + up + rt));
        packed[e] = c;
    }
}

// 4-corner image (dock.h: dock_grid.quad_dev): float4 [n_maps][ny][nx][nz].  A 32 (x) by 8 (z) tile goes through shared
// memory: rows of the plain maps are read along x, entries are written along z.  blockIdx.z = (system, map, z tile).
__global__ void __launch_bounds__(256) grid_quad_kernel(const GridSysArgs *__restrict__ sys, int n_maps, int zt_max)
{
    __shared__ float4 tile[32][9];
    const GridSysArgs S = sys[blockIdx.z / (n_maps * zt_max)];
    const int rem = blockIdx.z % (n_maps * zt_max), m = rem / zt_max, iz0 = (rem % zt_max) * 8, ix0 = blockIdx.x * 32, iy = blockIdx.y;
    const int nx = S.nx, ny = S.ny, nz = S.nz;
    if (!S.quad || iy >= ny || ix0 >= nx || iz0 >= nz) return;        // uniform per block
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    {
        const int ix = min(ix0 + tx, nx - 1), iz = min(iz0 + ty, nz - 1);
        const int ix1 = min(ix + 1, nx - 1), iy1 = min(iy + 1, ny - 1);
        const float *pl = S.out + ((size_t)m * nz + iz) * ny * nx;
        tile[tx][ty] = make_float4(pl[(size_t)iy * nx + ix], pl[(size_t)iy * nx + ix1], pl[(size_t)iy1 * nx + ix], pl[(size_t)iy1 * nx + ix1]);
    }
    __syncthreads();
    const int wx = threadIdx.x >> 3, wz = threadIdx.x & 7;
    if (ix0 + wx < nx && iz0 + wz < nz) S.quad[(((size_t)m * ny + iy) * nx + ix0 + wx) * nz + iz0 + wz] = tile[wx][wz];
}

struct GridPlan {
    int dims[3];
    float origin[3];
    float clo[3];
    int nc[3];
    float inv_cell;
    std::vector<float4> atoms;
    std::vector<int> cell_start;
    std::vector<float4> pair_tab;   // rows in processing order (maps sorted by ligand radius)
    int map_of[DOCK_MAX_XS_TYPES];
    unsigned fresh;
};

int plan_grid(const dock_params *p, const dock_protein *prot, const dock_box *box, int n_lig_types,
              const int32_t *lig_types, GridPlan &pl)
{
    if (dock_validate_params(p) != DOCK_OK || !prot || !box || !lig_types) return DOCK_EINVAL;
    if (prot->n < 0 || (prot->n > 0 && (!prot->xyz || !prot->type))) return DOCK_EINVAL;
    if (n_lig_types < 1 || n_lig_types > DOCK_MAX_XS_TYPES) return DOCK_EINVAL;
    if (dock_grid_dims(box, pl.dims) != DOCK_OK) return DOCK_EINVAL;
    for (int m = 0; m < n_lig_types; ++m)
        if (lig_types[m] < 0 || lig_types[m] >= p->n_types) return DOCK_EINVAL;
    for (int j = 0; j < prot->n; ++j)
        if (prot->type[j] < 0 || prot->type[j] >= p->n_types) return DOCK_EINVAL;
    const double cell = (double)p->cutoff + 0.01;   // edge > cutoff: a 1e-2 A guard band absorbs fp32 binning round-off
    double lo[3], hi[3];
    for (int c = 0; c < 3; ++c) {
        pl.origin[c] = (float)((double)box->center[c] - 0.5 * (double)box->size[c]);   // D-ORG: rounded once
        lo[c] = (double)pl.origin[c] - cell - 1e-3;
        hi[c] = (double)pl.origin[c] + (double)box->spacing * (pl.dims[c] - 1) + cell + 1e-3;
        pl.clo[c] = (float)lo[c];
        pl.nc[c] = (int)std::ceil((hi[c] - (double)pl.clo[c]) / cell);
        if (pl.nc[c] < 1) pl.nc[c] = 1;
    }
    const size_t ncells = (size_t)pl.nc[0] * pl.nc[1] * pl.nc[2];
    std::vector<int> cell_of(prot->n, -1), count(ncells + 1, 0);
    const float inv_cell = (float)(1.0 / cell);
    pl.inv_cell = inv_cell;
    for (int j = 0; j < prot->n; ++j) {
        int ci[3];
        bool inside = true;
        for (int c = 0; c < 3; ++c) {
            const float x = prot->xyz[3 * j + c];
            if (!(x >= pl.clo[c])) { inside = false; break; }
            ci[c] = (int)((x - pl.clo[c]) * inv_cell);
            if (ci[c] >= pl.nc[c]) { inside = false; break; }
        }
        if (!inside) continue;   // farther than the cutoff from every node
        cell_of[j] = (ci[2] * pl.nc[1] + ci[1]) * pl.nc[0] + ci[0];
        ++count[cell_of[j] + 1];
    }
    for (size_t c = 0; c < ncells; ++c) count[c + 1] += count[c];
    pl.cell_start = count;
    pl.atoms.assign(count[ncells] > 0 ? count[ncells] : 1, make_float4(0, 0, 0, 0));
    std::vector<int> cursor(count.begin(), count.end() - 1);
    for (int j = 0; j < prot->n; ++j) {
        if (cell_of[j] < 0) continue;
        float4 a = make_float4(prot->xyz[3 * j], prot->xyz[3 * j + 1], prot->xyz[3 * j + 2], 0.f);
        const int t = prot->type[j];
        std::memcpy(&a.w, &t, 4);
        pl.atoms[cursor[cell_of[j]]++] = a;
    }
    // processing order: maps sorted by ligand radius, so that maps of equal radius share the distance-only terms
    std::vector<int> order(n_lig_types);
    for (int m = 0; m < n_lig_types; ++m) order[m] = m;
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return p->radius[lig_types[a]] < p->radius[lig_types[b]]; });
    pl.fresh = 0u;
    pl.pair_tab.resize((size_t)n_lig_types * p->n_types);
    for (int k = 0; k < n_lig_types; ++k) {
        const int m = order[k], a = lig_types[m];
        pl.map_of[k] = m;
        if (k % MAPS_PER_PASS == 0 || p->radius[a] != p->radius[lig_types[order[k - 1]]]) pl.fresh |= 1u << k;
        for (int t = 0; t < p->n_types; ++t) {
            const float wh = (p->hydrophobic[a] && p->hydrophobic[t]) ? p->w[3] : 0.f;
            const float whb = ((p->donor[a] && p->acceptor[t]) || (p->donor[t] && p->acceptor[a])) ? p->w[4] : 0.f;
            pl.pair_tab[(size_t)k * p->n_types + t] = make_float4(p->radius[a] + p->radius[t], wh, whb, 0.f);
        }
    }
    return DOCK_OK;
}

}  // namespace

extern "C" int dock_grid_dims(const dock_box *box, int32_t dims[3])
{
    if (!box || !dims || !(box->spacing > 0.f)) return DOCK_EINVAL;
    for (int c = 0; c < 3; ++c) {
        if (!(box->size[c] > 0.f)) return DOCK_EINVAL;
        dims[c] = (int)std::floor((double)box->size[c] / (double)box->spacing + 0.5) + 1;
        if (dims[c] < 2 || dims[c] > 4096) return DOCK_EINVAL;
    }
    return DOCK_OK;
}

extern "C" size_t dock_grid_bytes(const dock_params *params, const dock_box *box, int32_t n_lig_types)
{
    int32_t dims[3];
    if (!params || n_lig_types < 1 || n_lig_types > DOCK_MAX_XS_TYPES || dock_grid_dims(box, dims) != DOCK_OK) return 0;
    const size_t ch = params->grad_mode == 1 ? 4 : 1;
    const size_t nodes = (size_t)dims[0] * dims[1] * dims[2] * (size_t)n_lig_types * ch;
    return align_up(nodes * sizeof(float), 256) + align_up(nodes * sizeof(Cell8), 256) + (ch == 1 ? nodes * sizeof(float4) : 0);
}

// All systems in ONE upload and two launches (build, pack): the per-system lattice descriptions, cell lists and sorted
// atoms are concatenated in the workspace; a block finds its system from GridSysArgs::block_begin.
extern "C" int dock_build_grids_batch(const dock_params *params, int32_t n_systems, const dock_protein *proteins,
                                      const dock_box *boxes, int32_t n_lig_types, const int32_t *lig_types,
                                      float *const *grid_dev, const size_t *grid_bytes, dock_grid *out_descs,
                                      void *ws_dev, size_t ws_bytes, size_t *needed, void *stream_)
{
    if (n_systems < 0 || (n_systems > 0 && (!proteins || !boxes))) return DOCK_EINVAL;
    if (n_systems == 0) {
        if (dock_validate_params(params) != DOCK_OK) return DOCK_EINVAL;
        if (needed) *needed = 0;
        return DOCK_OK;
    }
    std::vector<GridPlan> plans(n_systems);
    std::vector<GridSysArgs> sys(n_systems);
    size_t n_atoms = 0, n_cells = 0;
    long long n_blocks = 0;
    for (int s = 0; s < n_systems; ++s) {
        const int rc = plan_grid(params, &proteins[s], &boxes[s], n_lig_types, lig_types, plans[s]);
        if (rc != DOCK_OK) return rc;
        const GridPlan &pl = plans[s];
        GridSysArgs &S = sys[s];
        S.nx = pl.dims[0]; S.ny = pl.dims[1]; S.nz = pl.dims[2];
        S.ox = pl.origin[0]; S.oy = pl.origin[1]; S.oz = pl.origin[2];
        S.h = boxes[s].spacing;
        for (int c = 0; c < 3; ++c) S.clo[c] = pl.clo[c];
        S.inv_cell = pl.inv_cell;
        S.ncx = pl.nc[0]; S.ncy = pl.nc[1]; S.ncz = pl.nc[2];
        S.atoms_off = (int)n_atoms;
        S.cells_off = (int)n_cells;
        S.block_begin = (int)n_blocks;
        S.pad_ = 0;
        S.out = nullptr; S.packed = nullptr;
        n_atoms += pl.atoms.size();
        n_cells += pl.cell_start.size();
        n_blocks += (long long)((S.nx + 7) / 8) * ((S.ny + 7) / 8) * ((S.nz + 1) / 2);
        if (n_atoms > 0x7fffffffull || n_cells > 0x7fffffffull || n_blocks > 0x7fffffffLL) return DOCK_EINVAL;
    }
    const GridPlan &p0 = plans[0];                                      // the pair table depends on params and types only
    const size_t b_atoms = align_up(n_atoms * sizeof(float4), 256);
    const size_t b_cells = align_up(n_cells * sizeof(int), 256);
    const size_t b_tab = align_up(p0.pair_tab.size() * sizeof(float4), 256);
    const size_t b_sys = align_up((size_t)n_systems * sizeof(GridSysArgs), 256);
    const size_t need = b_atoms + b_cells + b_tab + b_sys;
    if (needed) *needed = need;
    if (!ws_dev || ws_bytes < need) return DOCK_EWORKSPACE;
    if (!grid_dev || !grid_bytes || !out_descs) return DOCK_EINVAL;
    const int channels = params->grad_mode == 1 ? 4 : 1;
    for (int s = 0; s < n_systems; ++s) {
        if (!grid_dev[s] || ((uintptr_t)grid_dev[s] & 255)) return DOCK_EINVAL;
        if (grid_bytes[s] < dock_grid_bytes(params, &boxes[s], n_lig_types)) return DOCK_EINVAL;   // buffer too small for the maps
        const size_t nodes = (size_t)sys[s].nx * sys[s].ny * sys[s].nz * (size_t)n_lig_types * channels;
        sys[s].out = grid_dev[s];
        sys[s].packed = reinterpret_cast<Cell8 *>(reinterpret_cast<unsigned char *>(grid_dev[s]) + align_up(nodes * sizeof(float), 256));
        sys[s].quad = channels == 1 ? reinterpret_cast<float4 *>(reinterpret_cast<unsigned char *>(sys[s].packed) + align_up(nodes * sizeof(Cell8), 256)) : nullptr;
    }
    // one host image, one copy
    std::vector<unsigned char> image(need, 0);
    for (int s = 0; s < n_systems; ++s) {
        std::memcpy(image.data() + (size_t)sys[s].atoms_off * sizeof(float4), plans[s].atoms.data(), plans[s].atoms.size() * sizeof(float4));
        std::memcpy(image.data() + b_atoms + (size_t)sys[s].cells_off * sizeof(int), plans[s].cell_start.data(), plans[s].cell_start.size() * sizeof(int));
    }
    std::memcpy(image.data() + b_atoms + b_cells, p0.pair_tab.data(), p0.pair_tab.size() * sizeof(float4));
    std::memcpy(image.data() + b_atoms + b_cells + b_tab, sys.data(), (size_t)n_systems * sizeof(GridSysArgs));
    cudaStream_t stream = (cudaStream_t)stream_;
    unsigned char *ws = (unsigned char *)ws_dev;
    DOCK_CUDA_CHECK(cudaMemcpyAsync(ws, image.data(), need, cudaMemcpyHostToDevice, stream));

    GridBuildArgs A;
    A.cutoff = params->cutoff;
    A.cutoff2 = params->cutoff * params->cutoff;
    A.n_maps = n_lig_types;
    A.n_types = params->n_types;
    for (int i = 0; i < 5; ++i) A.w[i] = params->w[i];
    A.atoms = (const float4 *)ws;
    A.cell_start = (const int *)(ws + b_atoms);
    A.pair_tab = (const float4 *)(ws + b_atoms + b_cells);
    A.channels = channels;
    for (int k = 0; k < DOCK_MAX_XS_TYPES; ++k) A.map_of[k] = k < n_lig_types ? p0.map_of[k] : 0;
    A.fresh = p0.fresh;
    A.sys = (const GridSysArgs *)(ws + b_atoms + b_cells + b_tab);
    A.n_sys = n_systems;
    dim3 grid((unsigned)n_blocks, (unsigned)((n_lig_types + MAPS_PER_PASS - 1) / MAPS_PER_PASS));
    if (channels == 4) grid_build_kernel<true><<<grid, 128, 0, stream>>>(A);
    else grid_build_kernel<false><<<grid, 128, 0, stream>>>(A);
    DOCK_LAUNCH_CHECK();
    const unsigned pack_x = (unsigned)std::max(1, std::min(148 * 16, 148 * 16 * 4 / n_systems + 1));
    grid_pack_kernel<<<dim3(pack_x, (unsigned)n_systems), 256, 0, stream>>>(A.sys, n_lig_types * channels);
    DOCK_LAUNCH_CHECK();
    if (channels == 1) {
        int mx = 0, my = 0, mz = 0;
        for (int s = 0; s < n_systems; ++s) { mx = std::max(mx, sys[s].nx); my = std::max(my, sys[s].ny); mz = std::max(mz, sys[s].nz); }
        const int zt = (mz + 7) / 8;
        // blockIdx.z = (system, map, z tile) is limited to 65535: as many systems per launch as fit (n_maps <= 32 and
        // zt <= 512, so one system always does; my <= 4096 by dock_grid_dims) -- nothing to reject here, after the enqueues
        const int per_launch = std::max(1, 65535 / (n_lig_types * zt));
        for (int s0 = 0; s0 < n_systems; s0 += per_launch) {
            const unsigned gz = (unsigned)(std::min(per_launch, n_systems - s0) * n_lig_types * zt);
            grid_quad_kernel<<<dim3((unsigned)((mx + 31) / 32), (unsigned)my, gz), 256, 0, stream>>>(A.sys + s0, n_lig_types, zt);
            DOCK_LAUNCH_CHECK();
        }
    }

    for (int s = 0; s < n_systems; ++s) {
        dock_grid *d = &out_descs[s];
        std::memset(d, 0, sizeof(*d));
        for (int c = 0; c < 3; ++c) { d->dims[c] = plans[s].dims[c]; d->origin[c] = plans[s].origin[c]; }
        d->spacing = boxes[s].spacing;
        d->n_maps = n_lig_types;
        for (int t = 0; t < DOCK_MAX_XS_TYPES; ++t) d->type_to_map[t] = -1;
        for (int m = 0; m < n_lig_types; ++m) d->type_to_map[lig_types[m]] = m;
        d->data_dev = grid_dev[s];
        d->packed_dev = reinterpret_cast<const float *>(sys[s].packed);
        d->n_channels = channels;
        d->quad_dev = reinterpret_cast<const float *>(sys[s].quad);
    }
    return DOCK_OK;
}

extern "C" int dock_build_grids(const dock_params *params, const dock_protein *protein, const dock_box *box,
                                int32_t n_lig_types, const int32_t *lig_types,
                                float *grid_dev, size_t grid_bytes, dock_grid *out_desc,
                                void *ws_dev, size_t ws_bytes, size_t *needed, void *stream_)
{
    if (!protein || !box) return DOCK_EINVAL;
    float *const gd[1] = {grid_dev};
    const size_t gb[1] = {grid_bytes};
    return dock_build_grids_batch(params, 1, protein, box, n_lig_types, lig_types, grid_dev ? gd : nullptr, gb, out_desc,
                                  ws_dev, ws_bytes, needed, stream_);
}
