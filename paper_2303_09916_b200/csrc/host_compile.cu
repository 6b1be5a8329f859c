// host_compile.cu -- parameter defaults, validation, and the ligand "compiler" (host only).
#include "host_compile.cuh"

#include <algorithm>
#include <cmath>
#include <cstring>

std::atomic<int> g_dock_last_cuda_error{0};
std::atomic<unsigned long long> g_dock_launches{0};

extern "C" int dock_last_cuda_error(void) { return g_dock_last_cuda_error.load(); }
extern "C" const char *dock_version(void) { return "dock_b200 0.2 (sm_100a)"; }
extern "C" uint64_t dock_launch_count(void) { return (uint64_t)g_dock_launches.load(); }

// Readings S1 (weights), S2 (XS radii / flags), S3, S7, S12, S14, S15, S19 of SURVEY.md 8(c): the paper
// prints none of these ("the same scoring function" as Vina).
extern "C" int dock_default_params(dock_params *p)
{
    if (!p) return DOCK_EINVAL;
    // id order: C_H C_P N_P N_D N_A N_DA O_P O_D O_A O_DA S_P P_P F_H Cl_H Br_H I_H Met_D
    static const float rad[17] = {1.9f, 1.9f, 1.8f, 1.8f, 1.8f, 1.8f, 1.7f, 1.7f, 1.7f, 1.7f,
                                  2.0f, 2.1f, 1.5f, 1.8f, 2.0f, 2.2f, 1.2f};
    static const int hyd[17] = {1, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 1, 1, 1, 1, 0};
    static const int don[17] = {0, 0, 0, 1, 0, 1, 0, 1, 0, 1, 0, 0, 0, 0, 0, 0, 1};
    static const int acc[17] = {0, 0, 0, 0, 1, 1, 0, 0, 1, 1, 0, 0, 0, 0, 0, 0, 0};
    std::memset(p, 0, sizeof(*p));
    p->n_types = 17;
    for (int i = 0; i < 17; ++i) {
        p->radius[i] = rad[i];
        p->hydrophobic[i] = hyd[i];
        p->donor[i] = don[i];
        p->acceptor[i] = acc[i];
    }
    p->w[0] = -0.0356f;
    p->w[1] = -0.00516f;
    p->w[2] = 0.840f;
    p->w[3] = -0.0351f;
    p->w[4] = -0.587f;
    p->cutoff = 8.0f;
    p->k_wall = 10.0f;
    p->t_mc = 1.2f;
    p->amp_trans = 2.0f;
    p->amp_rot = 0.3f;
    p->bfgs_c1 = 1e-4f;
    p->bfgs_shrink = 0.5f;
    p->bfgs_max_trials = 12;
    p->bfgs_gtol = 1e-3f;
    p->bfgs_curv_eps = 1e-8f;
    p->cluster_rmsd = 2.0f;
    p->topk = 10;
    p->optimizer = 0;
    p->bb_step = 1.0f;          // reading S13
    p->bb_fallback = 0.1f;
    p->grad_mode = 0;
    p->search_kernel = 0;
    p->score_kernel = 0;
    return DOCK_OK;
}

int dock_validate_params(const dock_params *p)
{
    if (!p) return DOCK_EINVAL;
    if (p->n_types <= 0 || p->n_types > DOCK_MAX_XS_TYPES) return DOCK_EINVAL;
    if (!(p->cutoff > 0.f) || !(p->t_mc > 0.f)) return DOCK_EINVAL;
    if (p->bfgs_max_trials < 1 || p->bfgs_max_trials > 64) return DOCK_EINVAL;
    if (!(p->bfgs_shrink > 0.f && p->bfgs_shrink < 1.f)) return DOCK_EINVAL;
    if (p->topk < 1 || p->topk > DOCK_MAX_TOPK) return DOCK_EINVAL;
    if (p->optimizer < 0 || p->optimizer > 1) return DOCK_EINVAL;
    if (p->grad_mode < 0 || p->grad_mode > 1) return DOCK_EINVAL;
    if (p->search_kernel < 0 || p->search_kernel > 2) return DOCK_EINVAL;
    if (p->score_kernel < 0 || p->score_kernel > 2) return DOCK_EINVAL;
    if (p->optimizer == 1 && (!(p->bb_step > 0.f) || !(p->bb_fallback > 0.f))) return DOCK_EINVAL;
    return DOCK_OK;
}

int dock_make_dev_params(const dock_params *p, DevParams *o)
{
    if (dock_validate_params(p) != DOCK_OK) return DOCK_EINVAL;
    for (int i = 0; i < 5; ++i) o->w[i] = p->w[i];
    o->cutoff = p->cutoff;
    o->cutoff2 = p->cutoff * p->cutoff;
    o->k_wall = p->k_wall;
    o->t_mc = p->t_mc;
    o->amp_trans = p->amp_trans;
    o->amp_rot = p->amp_rot;
    o->c1 = p->bfgs_c1;
    o->shrink = p->bfgs_shrink;
    o->gtol = p->bfgs_gtol;
    o->curv_eps = p->bfgs_curv_eps;
    o->max_trials = p->bfgs_max_trials;
    o->optimizer = p->optimizer;
    o->bb_step = p->bb_step;
    o->bb_fallback = p->bb_fallback;
    const double s1 = p->w[0] < 0.f ? -1.0 : 1.0, s2 = p->w[1] < 0.f ? -1.0 : 1.0;
    o->lw1 = p->w[0] != 0.f ? (float)std::log2(8.0 * std::fabs((double)p->w[0])) : -INFINITY;
    o->lw2 = p->w[1] != 0.f ? (float)std::log2(0.5 * std::fabs((double)p->w[1])) : -INFINITY;
    o->sigma = (float)-s1;
    o->q = (float)(s1 * s2);
    o->m3q = -3.f * o->q;
    o->c4 = o->sigma * 2.f * p->w[2];
    o->eA = (float)(s1 / 8.0);
    o->eB = (float)(2.0 * s2);
    return DOCK_OK;
}

int dock_make_dev_grid(const dock_params *p, const dock_grid *g, DevGrid *o)
{
    if (!p || !g || !g->data_dev || !g->packed_dev) return DOCK_EINVAL;
    if (g->dims[0] < 2 || g->dims[1] < 2 || g->dims[2] < 2 || !(g->spacing > 0.f)) return DOCK_EINVAL;
    if (g->n_maps < 1 || g->n_maps > DOCK_MAX_XS_TYPES) return DOCK_EINVAL;
    o->nx = g->dims[0]; o->ny = g->dims[1]; o->nz = g->dims[2];
    const double h = (double)g->spacing;
    int ic[3];
    float r32[3], rd[3];
    for (int c = 0; c < 3; ++c) {
        ic[c] = (g->dims[c] - 1) / 2;                                   // reference node near the centre
        const double r = (double)g->origin[c] + h * ic[c];              // its exact position
        r32[c] = (float)r;
        rd[c] = (float)(r - (double)r32[c]);
    }
    o->icx = ic[0]; o->icy = ic[1]; o->icz = ic[2];
    o->rx = r32[0]; o->ry = r32[1]; o->rz = r32[2];
    o->rdx = rd[0]; o->rdy = rd[1]; o->rdz = rd[2];
    o->lo_x = -(float)ic[0]; o->lo_y = -(float)ic[1]; o->lo_z = -(float)ic[2];
    o->hi_x = (float)(g->dims[0] - 1 - ic[0]); o->hi_y = (float)(g->dims[1] - 1 - ic[1]); o->hi_z = (float)(g->dims[2] - 1 - ic[2]);
    o->h = g->spacing;
    o->inv_h = (float)(1.0 / h);
    o->inv_h_lo = (float)(1.0 / h - (double)o->inv_h);
    o->kw_g = (float)(2.0 * (double)p->k_wall * h);
    o->kw_e = (float)((double)p->k_wall * h * h);
    if (g->n_channels != 0 && g->n_channels != 1 && g->n_channels != 4) return DOCK_EINVAL;
    o->channels = g->n_channels == 4 ? 4 : 1;
    o->chan_stride = g->dims[0] * g->dims[1] * g->dims[2];
    o->packed = reinterpret_cast<const Cell8 *>(g->packed_dev);
    o->data = g->data_dev;
    return DOCK_OK;
}

namespace {

template <class T>
size_t push_section(std::vector<unsigned char> &bytes, const std::vector<T> &v)
{
    size_t off = align_up(bytes.size(), 16);
    bytes.resize(off + std::max<size_t>(v.size() * sizeof(T), 16), 0);
    if (!v.empty()) std::memcpy(bytes.data() + off, v.data(), v.size() * sizeof(T));
    return off;
}

// Conflict-free pair schedule: every round holds <= 32 oriented pairs (src -> dst) whose sources
// are pairwise distinct atoms and whose destinations are pairwise distinct atoms, so the kernel can
// update g[src] for all lanes, then g[dst] for all lanes, with plain (non-atomic, deterministic)
// shared-memory read-modify-writes.
void build_schedule(const dock_params *p, const dock_ligand *L, std::vector<PairRec> &sched, int &n_rounds)
{
    struct E { int i, j; };
    std::vector<E> rem(L->P);
    for (int k = 0; k < L->P; ++k) rem[k] = {L->pairs[2 * k], L->pairs[2 * k + 1]};
    n_rounds = 0;
    sched.clear();
    std::vector<int> deg(L->N);
    std::vector<char> us(L->N), ud(L->N);
    while (!rem.empty()) {
        std::fill(deg.begin(), deg.end(), 0);
        for (const E &e : rem) { ++deg[e.i]; ++deg[e.j]; }
        std::stable_sort(rem.begin(), rem.end(), [&](const E &a, const E &b) {
            const int ka = std::max(deg[a.i], deg[a.j]) * 1000 + deg[a.i] + deg[a.j];
            const int kb = std::max(deg[b.i], deg[b.j]) * 1000 + deg[b.i] + deg[b.j];
            return ka > kb;
        });
        std::fill(us.begin(), us.end(), 0);
        std::fill(ud.begin(), ud.end(), 0);
        std::vector<E> keep, rnd;
        for (const E &e : rem) {
            if (rnd.size() < 32 && !us[e.i] && !ud[e.j]) { rnd.push_back({e.i, e.j}); us[e.i] = 1; ud[e.j] = 1; }
            else if (rnd.size() < 32 && !us[e.j] && !ud[e.i]) { rnd.push_back({e.j, e.i}); us[e.j] = 1; ud[e.i] = 1; }
            else keep.push_back(e);
        }
        for (int l = 0; l < 32; ++l) {
            PairRec r;
            if (l < (int)rnd.size()) {
                const int ti = L->type[rnd[l].i], tj = L->type[rnd[l].j];
                r.ij = rnd[l].i | (rnd[l].j << 16);
                r.rsum = p->radius[ti] + p->radius[tj];
                // wh' = -sigma w4, whb' = -sigma w5 / 0.7 (DevParams)
                const float sigma = p->w[0] < 0.f ? 1.f : -1.f;
                r.wh = (p->hydrophobic[ti] && p->hydrophobic[tj]) ? -sigma * p->w[3] : 0.f;
                r.whb = ((p->donor[ti] && p->acceptor[tj]) || (p->donor[tj] && p->acceptor[ti]))
                            ? (float)(-(double)sigma * (double)p->w[4] / 0.7) : 0.f;
            } else {
                r.ij = -1; r.rsum = TPP_MASKED_RSUM; r.wh = 0.f; r.whb = 0.f;
            }
            sched.push_back(r);
        }
        rem.swap(keep);
        ++n_rounds;
    }
}

}  // namespace

int dock_compile_ligand(const dock_params *p, const dock_grid *g, const dock_ligand *L, LigandBlob &out)
{
    if (!p || !L) return DOCK_EINVAL;
    const int N = L->N, T = L->T, P = L->P;
    if (N < 1 || N > DOCK_MAX_ATOMS || T < 0 || T > DOCK_MAX_TORSIONS || P < 0) return DOCK_EINVAL;
    if (!L->ref_xyz || !L->type || !L->atom_fragment) return DOCK_EINVAL;
    if (T > 0 && (!L->tors_parent || !L->tors_a || !L->tors_b)) return DOCK_EINVAL;
    if (P > 0 && !L->pairs) return DOCK_EINVAL;
    for (int i = 0; i < N; ++i) {
        const int t = L->type[i];
        if (t < 0 || t >= p->n_types) return DOCK_EINVAL;
        if (g && g->type_to_map[t] < 0) return DOCK_EINVAL;          // type without a map
        if (g && g->type_to_map[t] >= g->n_maps) return DOCK_EINVAL;
        if (L->atom_fragment[i] < 0 || L->atom_fragment[i] > T) return DOCK_EINVAL;
    }
    for (int k = 0; k < T; ++k) {
        if (L->tors_parent[k] < 0 || L->tors_parent[k] > k) return DOCK_EINVAL;      // parents first
        const int a = L->tors_a[k], b = L->tors_b[k];
        if (a < 0 || a >= N || b < 0 || b >= N || a == b) return DOCK_EINVAL;
        if (L->atom_fragment[a] != L->tors_parent[k]) return DOCK_EINVAL;            // axis atom in the wrong fragment
        if (L->atom_fragment[b] != k + 1) return DOCK_EINVAL;
    }
    {
        std::vector<unsigned char> seen((size_t)N * N, 0);
        for (int k = 0; k < P; ++k) {
            const int i = L->pairs[2 * k], j = L->pairs[2 * k + 1];
            if (i < 0 || i >= N || j < 0 || j >= N || i == j) return DOCK_EINVAL;
            const size_t key = (size_t)std::min(i, j) * N + std::max(i, j);
            if (seen[key]) return DOCK_EINVAL;                                       // a pair may be listed once
            seen[key] = 1;
        }
    }
    // pivot = centroid of the root-fragment reference atoms (reading S11), in double
    double c[3] = {0, 0, 0};
    int nroot = 0;
    for (int i = 0; i < N; ++i)
        if (L->atom_fragment[i] == 0) {
            for (int d = 0; d < 3; ++d) c[d] += (double)L->ref_xyz[3 * i + d];
            ++nroot;
        }
    if (nroot == 0) return DOCK_EINVAL;
    for (int d = 0; d < 3; ++d) c[d] /= nroot;

    const long long map_stride = g ? (long long)g->dims[0] * g->dims[1] * g->dims[2] : 0;
    std::vector<float4> atom_ref(N);
    std::vector<int2> atom_topo(N);
    for (int i = 0; i < N; ++i) {
        int mask = 0, f = L->atom_fragment[i];
        while (f > 0) { mask |= 1 << (f - 1); f = L->tors_parent[f - 1]; }
        const long long off = g ? (long long)g->type_to_map[L->type[i]] * map_stride * (g->n_channels == 4 ? 4 : 1) : 0;
        if (off > 0x7fffffffLL) return DOCK_EINVAL;
        atom_ref[i] = make_float4((float)((double)L->ref_xyz[3 * i] - c[0]), (float)((double)L->ref_xyz[3 * i + 1] - c[1]),
                                  (float)((double)L->ref_xyz[3 * i + 2] - c[2]), 0.f);
        const int ioff = (int)off;
        std::memcpy(&atom_ref[i].w, &ioff, 4);
        atom_topo[i] = make_int2(L->atom_fragment[i], mask);
    }
    std::vector<float4> tors_axis(T), tors_pt(T);
    std::vector<int2> tors_ab(T);
    for (int k = 0; k < T; ++k) {
        const int a = L->tors_a[k], b = L->tors_b[k];
        double u[3], n = 0;
        for (int d = 0; d < 3; ++d) { u[d] = (double)L->ref_xyz[3 * b + d] - (double)L->ref_xyz[3 * a + d]; n += u[d] * u[d]; }
        n = std::sqrt(n);
        if (!(n > 1e-6)) return DOCK_EINVAL;
        tors_axis[k] = make_float4((float)(u[0] / n), (float)(u[1] / n), (float)(u[2] / n), 0.f);
        tors_pt[k] = make_float4((float)((double)L->ref_xyz[3 * b] - c[0]), (float)((double)L->ref_xyz[3 * b + 1] - c[1]),
                                 (float)((double)L->ref_xyz[3 * b + 2] - c[2]), 0.f);
        const int par = L->tors_parent[k];
        std::memcpy(&tors_pt[k].w, &par, 4);
        tors_ab[k] = make_int2(a, b);
    }
    std::vector<PairRec> sched;
    int n_rounds = 0;
    build_schedule(p, L, sched, n_rounds);

    out.bytes.clear();
    DevLigand &r = out.rel;
    r.N = N; r.T = T; r.P = P; r.n_rounds = n_rounds;
    r.n_pad = (N + 3) & ~3;
    r.atom_ref = (const float4 *)push_section(out.bytes, atom_ref);
    r.atom_topo = (const int2 *)push_section(out.bytes, atom_topo);
    r.tors_axis = (const float4 *)push_section(out.bytes, tors_axis);
    r.tors_pt = (const float4 *)push_section(out.bytes, tors_pt);
    r.tors_ab = (const int2 *)push_section(out.bytes, tors_ab);
    r.sched = (const PairRec *)push_section(out.bytes, sched);
    out.bytes.resize(align_up(out.bytes.size(), 256), 0);
    return DOCK_OK;
}

DevLigand dock_relocate_ligand(const LigandBlob &b, const unsigned char *base)
{
    DevLigand d = b.rel;
    d.atom_ref = (const float4 *)(base + (size_t)b.rel.atom_ref);
    d.atom_topo = (const int2 *)(base + (size_t)b.rel.atom_topo);
    d.tors_axis = (const float4 *)(base + (size_t)b.rel.tors_axis);
    d.tors_pt = (const float4 *)(base + (size_t)b.rel.tors_pt);
    d.tors_ab = (const int2 *)(base + (size_t)b.rel.tors_ab);
    d.sched = (const PairRec *)(base + (size_t)b.rel.sched);
    return d;
}

// ---- thread-per-pose tables ------------------------------------------------------------------------
int dock_compile_tpp(const dock_params *p, const dock_grid *g, const dock_ligand *L, TppLigand &out,
                     std::vector<uint4> &overflow)
{
    LigandBlob chk;                                   // reuse the validation of the warp-per-pose compiler
    if (!g || dock_compile_ligand(p, g, L, chk) != DOCK_OK) return DOCK_EINVAL;
    const int N = L->N, T = L->T, P = L->P;
    std::memset(&out, 0, sizeof(out));
    overflow.clear();
    out.N = N; out.T = T;

    double c[3] = {0, 0, 0};
    int nroot = 0;
    for (int i = 0; i < N; ++i)
        if (L->atom_fragment[i] == 0) {
            for (int d = 0; d < 3; ++d) c[d] += (double)L->ref_xyz[3 * i + d];
            ++nroot;
        }
    for (int d = 0; d < 3; ++d) c[d] /= nroot;

    // slots = atoms sorted by fragment (stable), so that a fragment's atoms are contiguous
    std::vector<int> atom_of(N), slot_of(N);
    for (int i = 0; i < N; ++i) atom_of[i] = i;
    std::stable_sort(atom_of.begin(), atom_of.end(),
                     [&](int a, int b) { return L->atom_fragment[a] < L->atom_fragment[b]; });
    for (int s = 0; s < N; ++s) slot_of[atom_of[s]] = s;
    const long long map_stride = (long long)g->dims[0] * g->dims[1] * g->dims[2];
    int f_cur = 0;
    for (int s = 0; s < N; ++s) {
        const int i = atom_of[s];
        const long long off = (long long)g->type_to_map[L->type[i]] * map_stride * (g->n_channels == 4 ? 4 : 1);
        if (off > 0x7fffffffLL) return DOCK_EINVAL;
        const int ioff = (int)off;
        out.atom_ref[s] = make_float4((float)((double)L->ref_xyz[3 * i] - c[0]), (float)((double)L->ref_xyz[3 * i + 1] - c[1]),
                                      (float)((double)L->ref_xyz[3 * i + 2] - c[2]), 0.f);
        std::memcpy(&out.atom_ref[s].w, &ioff, 4);
        while (f_cur < L->atom_fragment[i]) out.frag_end[f_cur++] = (unsigned char)s;
    }
    while (f_cur <= T) out.frag_end[f_cur++] = (unsigned char)N;
    // fragment f's sums may overwrite the force slots 2(f-1), 2(f-1)+1 iff those atoms were consumed before: frag_end[f] >= 2f
    out.fm_alias = 1;
    for (int f = 1; f <= T; ++f)
        if ((int)out.frag_end[f] < 2 * f) out.fm_alias = 0;
    for (int k = 0; k < T; ++k) {
        const int a = L->tors_a[k], b = L->tors_b[k];
        double u[3], n = 0;
        for (int d = 0; d < 3; ++d) { u[d] = (double)L->ref_xyz[3 * b + d] - (double)L->ref_xyz[3 * a + d]; n += u[d] * u[d]; }
        n = std::sqrt(n);
        const int par = L->tors_parent[k];
        out.tors_axis[k] = make_float4((float)(u[0] / n), (float)(u[1] / n), (float)(u[2] / n), 0.f);
        std::memcpy(&out.tors_axis[k].w, &par, 4);
        out.tors_pt[k] = make_float4((float)((double)L->ref_xyz[3 * b] - c[0]), (float)((double)L->ref_xyz[3 * b + 1] - c[1]),
                                     (float)((double)L->ref_xyz[3 * b + 2] - c[2]), (float)(1.0 / n));
        out.tors_a[k] = (unsigned char)slot_of[a];
        out.tors_b[k] = (unsigned char)slot_of[b];
    }

    // pair schedule: tiles of TPP_TILE consecutive slots.  The pairs between two tiles A < B form a
    // small bit matrix; they all go either to A's group (one record per partner j in B) or to B's
    // group (one record per partner j in A), whichever needs fewer records.  Format: common.cuh.
    const int n_tiles = (N + TPP_TILE - 1) / TPP_TILE;
    const float sigma = p->w[0] < 0.f ? 1.f : -1.f;                 // DevParams::sigma
    const float whp = -sigma * p->w[3];                             // wh'
    const float whbp = (float)(-(double)sigma * (double)p->w[4] / 0.7);   // whb'
    struct Rec { int j; int cls; float rsum[TPP_TILE], wh[TPP_TILE], whb[TPP_TILE]; };
    std::vector<std::vector<Rec>> groups(n_tiles);
    std::vector<std::vector<std::pair<int, int>>> between((size_t)n_tiles * n_tiles);   // (slot in A, slot in B)
    for (int k = 0; k < P; ++k) {
        int sa = slot_of[L->pairs[2 * k]], sb = slot_of[L->pairs[2 * k + 1]];
        if (sa > sb) std::swap(sa, sb);
        between[(size_t)(sa / TPP_TILE) * n_tiles + sb / TPP_TILE].push_back({sa, sb});
    }
    auto add = [&](int tile, int i_slot, int j_slot) {
        std::vector<Rec> &grp = groups[tile];
        Rec *r = nullptr;
        for (Rec &q : grp) if (q.j == j_slot) { r = &q; break; }
        if (!r) {
            Rec fresh;
            fresh.j = j_slot;
            fresh.cls = 0;
            for (int t = 0; t < TPP_TILE; ++t) { fresh.rsum[t] = -TPP_MASKED_RSUM; fresh.wh[t] = 0.f; fresh.whb[t] = 0.f; }   // rsum[] holds -(R_i+R_j)
            grp.push_back(fresh);
            r = &grp.back();
        }
        const int t = i_slot - tile * TPP_TILE;
        const int ti = L->type[atom_of[i_slot]], tj = L->type[atom_of[j_slot]];
        r->rsum[t] = -(p->radius[ti] + p->radius[tj]);
        if (p->hydrophobic[ti] && p->hydrophobic[tj] && p->w[3] != 0.f) { r->wh[t] = whp; r->cls = std::max(r->cls, 1); }
        if (((p->donor[ti] && p->acceptor[tj]) || (p->donor[tj] && p->acceptor[ti])) && p->w[4] != 0.f) { r->whb[t] = whbp; r->cls = 2; }
    };
    for (int A = 0; A < n_tiles; ++A)
        for (int B = A; B < n_tiles; ++B) {
            const auto &pl = between[(size_t)A * n_tiles + B];
            if (pl.empty()) continue;
            uint32_t rows = 0, cols = 0;
            for (auto &e : pl) { rows |= 1u << (e.first - A * TPP_TILE); cols |= 1u << (e.second - B * TPP_TILE); }
            const bool to_a = (A == B) || __builtin_popcount(cols) <= __builtin_popcount(rows);
            for (auto &e : pl) {
                if (to_a) add(A, e.first, e.second);
                else add(B, e.second, e.first);
            }
        }
    std::vector<uint4> quads;
    auto fq = [](const float *v) {
        uint4 q;
        std::memcpy(&q, v, 16);
        return q;
    };
    for (int A = 0; A < n_tiles; ++A) {
        std::vector<Rec> &grp = groups[A];
        std::stable_sort(grp.begin(), grp.end(), [](const Rec &a, const Rec &b) { return a.j < b.j; });
        std::vector<const Rec *> cls[3];
        for (const Rec &r : grp) cls[r.cls].push_back(&r);
        const int n_i = std::min(TPP_TILE, N - A * TPP_TILE);
        uint4 hdr = make_uint4(0u, 0u, 0u, 0u);
        for (int t = 0; t < TPP_TILE; ++t) hdr.x |= (uint32_t)(A * TPP_TILE + (t < n_i ? t : 0)) << (8 * t);
        hdr.y = (uint32_t)(cls[0].size() / 2) | ((uint32_t)(cls[0].size() & 1) << 8) |
                ((uint32_t)(cls[1].size() / 2) << 16) | ((uint32_t)(cls[1].size() & 1) << 24);
        hdr.z = (uint32_t)(cls[2].size() / 2) | ((uint32_t)(cls[2].size() & 1) << 8) | ((uint32_t)n_i << 16);
        quads.push_back(hdr);
        for (int c = 0; c < 3; ++c) {
            const std::vector<const Rec *> &v = cls[c];
            auto payload = [&](const Rec *r) {
                quads.push_back(fq(r->rsum));
                if (c >= 1) quads.push_back(fq(r->wh));
                if (c >= 2) quads.push_back(fq(r->whb));
            };
            size_t k = 0;
            for (; k + 1 < v.size(); k += 2) {
                quads.push_back(make_uint4((uint32_t)v[k]->j * 128u, (uint32_t)v[k + 1]->j * 128u, 0u, 0u));
                payload(v[k]);
                payload(v[k + 1]);
            }
            if (k < v.size()) {
                quads.push_back(make_uint4((uint32_t)v[k]->j * 128u, 0u, 0u, 0u));
                payload(v[k]);
            }
        }
    }
    const int n_groups = n_tiles;
    out.n_groups = n_groups;
    if (quads.size() <= (size_t)TPP_SCHED_QUADS) {
        out.sched_in_param = 1;
        if (!quads.empty()) std::memcpy(out.sched, quads.data(), quads.size() * sizeof(uint4));
    } else {
        out.sched_in_param = 0;
        overflow.swap(quads);
    }
    return DOCK_OK;
}
