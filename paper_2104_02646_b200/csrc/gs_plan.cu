// gs_plan.cu -- host preprocessing of a scene: validation, rest-shape quantities, Morton reordering of
// particles and elements, tiling with tile-local indices and per-tile gather lists, upload into the
// caller's workspace.  Off the hot path (runs once per model).
//
// Rest quantities (fp64 on the host, stored fp32):
//   tets      B = D_m^-1, V = det(D_m)/6                         PAPER.md:575-581 (V_e, constant-strain tets)
//   triangles 2x2 B in the rest frame (t1, t2), A = det(D_m)/2   PAPER.md:584; A4
//   hinges    theta0 (signed rest dihedral), l0 (rest edge)      PAPER.md:585-586; A5, A6
#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <numeric>

#include "gs_internal.h"

namespace gs {

static thread_local char t_err[512] = "";
std::atomic<uint64_t> g_launches{0};
thread_local bool t_capturing = false;
thread_local uint64_t t_captured = 0;

void set_error(const char *fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(t_err, sizeof t_err, fmt, ap);
    va_end(ap);
}
const char *last_error() { return t_err; }
int cuda_fail(cudaError_t e, const char *what) {
    set_error("%s: %s", what, cudaGetErrorString(e));
    return GS_ECUDA;
}

// ---------------------------------------------------------------------------------- workspace layout
struct Bump {
    char *base;
    size_t off = 0;
    explicit Bump(void *b) : base((char *)b) {}
    template <class T>
    T *take(size_t n) {
        off = (off + 255) & ~(size_t)255;
        T *p = base ? (T *)(base + off) : nullptr;
        off += (n ? n : 1) * sizeof(T);
        return p;
    }
};

struct Layout {
    // per type
    char *rec[N_TYPES];
    int *tile_parts[N_TYPES], *perm[N_TYPES], *det[N_TYPES];
    float *par[N_TYPES], *g32[N_TYPES];
    double *g64[N_TYPES];
    int *perm_p, *bad;
    float *inv_mass, *gmass32, *ke, *kd, *kf, *muc, *kdrag, *klift;
    double *gmass64, *gcon64, *gacc;
    int *tile_ctr;
    const float **frame_base;
    float4 *f, *xs[2], *vs[2], *adjx, *adjv, *adjf;
    size_t bytes;
};

static Layout make_layout(void *base, int N, int E, const int counts[N_TYPES]) {
    Layout L;
    Bump b(base);
    const size_t EN = (size_t)E * N;
    for (int t = 0; t < N_TYPES; t++) {
        const size_t c = counts[t], a = kArity[t], nt = (c + kTileElems - 1) / kTileElems, cp = nt * kTileElems;
        // upper bounds (pmax <= arity * kTileElems is only known after the mesh has been tiled)
        L.rec[t] = b.take<char>(nt * (size_t)rec_bytes_of(t));
        L.tile_parts[t] = b.take<int>(2 * a * cp);  // 6 bytes per entry (id + local index), upper bound
        if (t != T_HINGE) {
            L.par[t] = b.take<float>(3 * E * cp);
            L.g32[t] = b.take<float>(kNumGrads[t] * E * cp);
            L.g64[t] = b.take<double>(kNumGrads[t] * E * cp);
        } else {
            L.par[t] = nullptr;
            L.g32[t] = b.take<float>(E * cp);
            L.g64[t] = b.take<double>(E * cp);
        }
        L.perm[t] = b.take<int>(c);
        L.det[t] = b.take<int>(nt);
    }
    L.perm_p = b.take<int>(N);
    L.inv_mass = b.take<float>(EN);
    L.gmass32 = b.take<float>(EN);
    L.gmass64 = b.take<double>(EN);
    L.gacc = b.take<double>((size_t)E * kConSlots * kAccVals);
    L.gcon64 = b.take<double>((size_t)E * kAccVals);
    L.tile_ctr = b.take<int>(8);
    L.frame_base = b.take<const float *>(1);
    L.ke = b.take<float>(E); L.kd = b.take<float>(E); L.kf = b.take<float>(E); L.muc = b.take<float>(E);
    L.kdrag = b.take<float>(E); L.klift = b.take<float>(E);
    L.bad = b.take<int>(1);
    L.f = b.take<float4>(EN);
    for (int i = 0; i < 2; i++) { L.xs[i] = b.take<float4>(EN); L.vs[i] = b.take<float4>(EN); }
    L.adjx = b.take<float4>(EN); L.adjv = b.take<float4>(EN); L.adjf = b.take<float4>(EN);
    L.bytes = ((b.off + 255) & ~(size_t)255) + 256;
    return L;
}

size_t workspace_bytes_upper(int N, int E, const int counts[N_TYPES]) { return make_layout(nullptr, N, E, counts).bytes; }

// ---------------------------------------------------------------------------------- geometry helpers (fp64)
struct d3 { double x, y, z; };
static inline d3 sub(d3 a, d3 b) { return {a.x - b.x, a.y - b.y, a.z - b.z}; }
static inline d3 crs(d3 a, d3 b) { return {a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x}; }
static inline double dt3(d3 a, d3 b) { return a.x * b.x + a.y * b.y + a.z * b.z; }
static inline d3 scl(double s, d3 a) { return {s * a.x, s * a.y, s * a.z}; }
static inline d3 P(const float *x, int i) { return {x[3 * i], x[3 * i + 1], x[3 * i + 2]}; }

static inline uint64_t spread21(uint64_t v) {
    v &= 0x1fffff;
    v = (v | v << 32) & 0x1f00000000ffffULL;
    v = (v | v << 16) & 0x1f0000ff0000ffULL;
    v = (v | v << 8) & 0x100f00f00f00f00fULL;
    v = (v | v << 4) & 0x10c30c30c30c30c3ULL;
    v = (v | v << 2) & 0x1249249249249249ULL;
    return v;
}

template <class T>
static int upload(T *dst, const std::vector<T> &src, cudaStream_t st) {
    if (src.empty()) return GS_OK;
    cudaError_t e = cudaMemcpyAsync(dst, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice, st);
    return e == cudaSuccess ? GS_OK : cuda_fail(e, "upload");
}
#define UP(dst, vec) do { int rc_ = upload(dst, vec, stream); if (rc_ != GS_OK) return rc_; } while (0)

// ---------------------------------------------------------------------------------- build
int build_model(const gs_model_desc *d, void *d_workspace, size_t bytes, cudaStream_t stream, gs_model *m) {
    const int N = d->n_particles, E = d->n_envs;
    const int counts[N_TYPES] = {d->n_tets, d->n_tris, d->n_hinges};
    Layout L = make_layout(d_workspace, N, E, counts);
    if (bytes < L.bytes) { set_error("workspace too small: %zu < %zu bytes", bytes, L.bytes); return GS_EINVAL; }
    if (((uintptr_t)d_workspace & 255) != 0) { set_error("workspace must be 256-byte aligned"); return GS_EINVAL; }
    const float *X = d->x_rest;

    // ---- validation of indices and masses
    const int32_t *conn[N_TYPES] = {d->tets, d->tris, d->hinges};
    static const char *tname[N_TYPES] = {"tet", "triangle", "hinge"};
    for (int t = 0; t < N_TYPES; t++)
        for (int e = 0; e < counts[t]; e++)
            for (int k = 0; k < kArity[t]; k++) {
                int i = conn[t][(size_t)e * kArity[t] + k];
                if (i < 0 || i >= N) { set_error("%s %d: particle index %d out of range [0, %d)", tname[t], e, i, N); return GS_EMESH; }
                for (int q = 0; q < k; q++)
                    if (conn[t][(size_t)e * kArity[t] + q] == i) { set_error("%s %d: repeated particle index %d", tname[t], e, i); return GS_EMESH; }
            }
    const size_t n_mass = (d->param_layout & GS_MASS_PER_ENV) ? (size_t)E * N : (size_t)N;
    for (size_t i = 0; i < n_mass; i++)
        if (!(d->mass[i] > 0.0f) || !std::isfinite(d->mass[i])) { set_error("mass[%zu] must be finite and > 0", i); return GS_EINVAL; }
    for (int i = 0; i < 3 * N; i++)
        if (!std::isfinite(X[i])) { set_error("x_rest has a non-finite entry at particle %d", i / 3); return GS_EINVAL; }

    // ---- particle Morton order
    double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300};
    for (int i = 0; i < N; i++)
        for (int r = 0; r < 3; r++) { lo[r] = std::min(lo[r], (double)X[3 * i + r]); hi[r] = std::max(hi[r], (double)X[3 * i + r]); }
    double span = 1e-30;
    for (int r = 0; r < 3; r++) span = std::max(span, hi[r] - lo[r]);
    auto morton = [&](double x, double y, double z) -> uint64_t {
        const double s = 2097151.0 / span;
        uint64_t ix = (uint64_t)std::min(2097151.0, std::max(0.0, (x - lo[0]) * s));
        uint64_t iy = (uint64_t)std::min(2097151.0, std::max(0.0, (y - lo[1]) * s));
        uint64_t iz = (uint64_t)std::min(2097151.0, std::max(0.0, (z - lo[2]) * s));
        return spread21(ix) | (spread21(iy) << 1) | (spread21(iz) << 2);
    };
    std::vector<uint64_t> key(N);
    for (int i = 0; i < N; i++) key[i] = morton(X[3 * i], X[3 * i + 1], X[3 * i + 2]);
    m->perm_p.resize(N);
    std::iota(m->perm_p.begin(), m->perm_p.end(), 0);
    std::stable_sort(m->perm_p.begin(), m->perm_p.end(), [&](int a, int b) { return key[a] < key[b]; });
    std::vector<int> inv_p(N);  // caller -> internal
    for (int i = 0; i < N; i++) inv_p[m->perm_p[i]] = i;
    UP(L.perm_p, m->perm_p);

    // ---- per-particle parameters
    {
        std::vector<float> w((size_t)E * N);
        for (int env = 0; env < E; env++)
            for (int i = 0; i < N; i++) {
                int c = m->perm_p[i];
                float mass = (d->param_layout & GS_MASS_PER_ENV) ? d->mass[(size_t)env * N + c] : d->mass[c];
                w[(size_t)env * N + i] = (d->pinned && d->pinned[c]) ? 0.0f : 1.0f / mass;
            }
        UP(L.inv_mass, w);
        std::vector<float> s(E);
        const float *src[4] = {d->ke, d->kd, d->kf, d->mu_c};
        float *dst[4] = {L.ke, L.kd, L.kf, L.muc};
        for (int q = 0; q < 4; q++) {
            for (int env = 0; env < E; env++) s[env] = (d->param_layout & GS_CONTACT_PER_ENV) ? src[q][env] : src[q][0];
            UP(dst[q], s);
        }
        const float *asrc[2] = {d->k_drag, d->k_lift};
        float *adst[2] = {L.kdrag, L.klift};
        m->aero_host = false;
        for (int q = 0; q < 2; q++) {
            for (int env = 0; env < E; env++) {
                s[env] = asrc[q] ? ((d->param_layout & GS_CONTACT_PER_ENV) ? asrc[q][env] : asrc[q][0]) : 0.0f;
                if (!std::isfinite(s[env]) || s[env] < 0.0f) { set_error("k_drag / k_lift must be finite and >= 0"); return GS_EINVAL; }
                if (s[env] != 0.0f) m->aero_host = true;
            }
            UP(adst[q], s);
        }
    }

    // ---- elements: rest quantities, Morton order, tiles
    ModelDev &dev = m->dev;
    memset(&dev, 0, sizeof dev);
    std::vector<std::vector<int>> all_tids[N_TYPES];  // particles of every tile, kept for the tile colouring below
    for (int t = 0; t < N_TYPES; t++) {
        const int c = counts[t], a = kArity[t];
        const int nt = (c + kTileElems - 1) / kTileElems;
        HostElemSet &hs = m->hes[t];
        hs.count = c; hs.n_tiles = nt; hs.max_tile_parts = 0;
        hs.perm.resize(c);
        std::vector<uint64_t> ekey(c);
        // rest quantities in caller order first
        std::vector<float4> r0(c), r1(c);
        std::vector<float2> r2(c);
        for (int e = 0; e < c; e++) {
            const int32_t *ix = conn[t] + (size_t)e * a;
            d3 cen = {0, 0, 0};
            for (int k = 0; k < a; k++) { d3 p = P(X, ix[k]); cen.x += p.x / a; cen.y += p.y / a; cen.z += p.z / a; }
            ekey[e] = morton(cen.x, cen.y, cen.z);
            if (t == T_TET) {
                d3 x0 = P(X, ix[0]), e1 = sub(P(X, ix[1]), x0), e2 = sub(P(X, ix[2]), x0), e3 = sub(P(X, ix[3]), x0);
                // D_m columns e1 e2 e3; inverse rows = (e2 x e3, e3 x e1, e1 x e2) / det
                d3 r_0 = crs(e2, e3), r_1 = crs(e3, e1), r_2 = crs(e1, e2);
                double det = dt3(e1, r_0);
                if (!(det > 0.0) || !std::isfinite(det)) { set_error("tet %d: non-positive rest volume (det D_m = %g)", e, det); return GS_EMESH; }
                r_0 = scl(1.0 / det, r_0); r_1 = scl(1.0 / det, r_1); r_2 = scl(1.0 / det, r_2);
                r0[e] = make_float4((float)r_0.x, (float)r_0.y, (float)r_0.z, (float)r_1.x);
                r1[e] = make_float4((float)r_1.y, (float)r_1.z, (float)r_2.x, (float)r_2.y);
                r2[e] = make_float2((float)r_2.z, (float)(det / 6.0));
            } else if (t == T_TRI) {
                d3 x0 = P(X, ix[0]), e1 = sub(P(X, ix[1]), x0), e2 = sub(P(X, ix[2]), x0), nn = crs(e1, e2);
                double l1 = std::sqrt(dt3(e1, e1)), ln = std::sqrt(dt3(nn, nn));
                if (!(0.5 * ln > 1e-12) || !(l1 > 0)) { set_error("triangle %d: degenerate rest shape (area %g)", e, 0.5 * ln); return GS_EMESH; }
                d3 t1 = scl(1.0 / l1, e1), t2 = crs(scl(1.0 / ln, nn), t1);
                double A = dt3(t1, e1), B = dt3(t1, e2), C = dt3(t2, e1), D = dt3(t2, e2), det = A * D - B * C;
                r0[e] = make_float4((float)(D / det), (float)(-B / det), (float)(-C / det), (float)(A / det));
                r1[e] = make_float4((float)(det / 2.0), 0.f, 0.f, 0.f);
            } else {
                d3 x1 = P(X, ix[0]), x2 = P(X, ix[1]), x3 = P(X, ix[2]), x4 = P(X, ix[3]);
                d3 n1 = crs(sub(x1, x3), sub(x1, x4)), n2 = crs(sub(x2, x4), sub(x2, x3)), ed = sub(x4, x3);
                double l0 = std::sqrt(dt3(ed, ed)), a1 = std::sqrt(dt3(n1, n1)), a2 = std::sqrt(dt3(n2, n2));
                if (!(l0 > 0) || !(a1 > 1e-12) || !(a2 > 1e-12)) { set_error("hinge %d: degenerate rest shape", e); return GS_EMESH; }
                d3 eh = scl(1.0 / l0, ed);
                double th = std::atan2(dt3(crs(scl(1 / a1, n1), scl(1 / a2, n2)), eh), dt3(n1, n2) / (a1 * a2));
                r0[e] = make_float4((float)std::sin(0.5 * th), (float)std::cos(0.5 * th), (float)((double)d->hinge_kb[e] * l0), (float)l0);
            }
        }
        std::iota(hs.perm.begin(), hs.perm.end(), 0);
        std::stable_sort(hs.perm.begin(), hs.perm.end(), [&](int x, int y) { return ekey[x] < ekey[y]; });
        const int cp = nt * kTileElems;
        hs.cpad = cp;
        // tiles, pass 1: the particles of each tile and the fullest tile
        std::vector<std::vector<int>> tids(nt);
        std::vector<std::vector<int>> tcnt(nt);
        std::vector<int> ids, cnt, order;
        for (int j = 0; j < nt; j++) {
            const int e0 = j * kTileElems, e1 = std::min(c, e0 + kTileElems);
            ids.clear();
            for (int e = e0; e < e1; e++)
                for (int k = 0; k < a; k++) ids.push_back(inv_p[conn[t][(size_t)hs.perm[e] * a + k]]);
            std::sort(ids.begin(), ids.end());
            std::vector<int> uniq, ucnt;
            for (size_t q = 0; q < ids.size();) {
                size_t q1 = q;
                while (q1 < ids.size() && ids[q1] == ids[q]) q1++;
                uniq.push_back(ids[q]); ucnt.push_back((int)(q1 - q));
                q = q1;
            }
            order.resize(uniq.size());
            std::iota(order.begin(), order.end(), 0);
            // ascending internal (Morton) id: the lanes of a warp gather neighbouring particles, i.e. few distinct 128-byte
            // lines per cp.async instruction (measured: 18 L1 wavefronts per gather instruction with a valence-sorted list)
            tids[j].resize(uniq.size()); tcnt[j].resize(uniq.size());
            for (size_t q = 0; q < uniq.size(); q++) { tids[j][q] = uniq[order[q]]; tcnt[j][q] = ucnt[order[q]]; }
            hs.max_tile_parts = std::max(hs.max_tile_parts, (int)uniq.size());
        }
        const int pmax = std::max(8, (hs.max_tile_parts + 7) / 8 * 8);
        hs.pmax = pmax;
        // pass 1b: tile-local indices by greedy 8-colouring.  An LDS.128 is served a quarter-warp (8 lanes) at a time and is
        // conflict-free when the 8 lanes hit 8 different 16-byte bank groups, i.e. local indices with different
        // residues mod 8 (or the same index: broadcast).  Particles that one quarter-warp reads for the same vertex
        // position therefore get different colours; colour c owns the local indices c, c + 8, c + 16, ...
        std::vector<std::vector<int>> tloc(nt);
        int lmax = 8;
        {
            std::vector<int> colour, seen_mask, csize(8);
            for (int j = 0; j < nt; j++) {
                const int e0 = j * kTileElems, e1 = std::min(c, e0 + kTileElems), P_ = (int)tids[j].size();
                auto local_of = [&](int gi) { return (int)(std::lower_bound(tids[j].begin(), tids[j].end(), gi) - tids[j].begin()); };
                // groups[(quarter, k)] = distinct list positions
                const int nq = (e1 - e0 + 7) / 8;
                std::vector<std::vector<int>> groups((size_t)nq * a), of_part(P_);
                for (int e = e0; e < e1; e++)
                    for (int k = 0; k < a; k++) {
                        const int q = local_of(inv_p[conn[t][(size_t)hs.perm[e] * a + k]]), g = ((e - e0) / 8) * a + k;
                        if (std::find(groups[g].begin(), groups[g].end(), q) == groups[g].end()) { groups[g].push_back(q); of_part[q].push_back(g); }
                    }
                colour.assign(P_, -1);
                std::fill(csize.begin(), csize.end(), 0);
                const int cap = (P_ + 7) / 8 + 1;  // bound the imbalance: lmax <= pmax + 16
                for (int e = e0; e < e1; e++)
                    for (int k = 0; k < a; k++) {
                        const int q = local_of(inv_p[conn[t][(size_t)hs.perm[e] * a + k]]);
                        if (colour[q] >= 0) continue;
                        unsigned forbid = 0;
                        for (int g : of_part[q])
                            for (int r : groups[g])
                                if (colour[r] >= 0) forbid |= 1u << colour[r];
                        int best = -1;
                        for (int cc = 0; cc < 8; cc++)
                            if (!(forbid >> cc & 1u) && csize[cc] < cap && (best < 0 || csize[cc] < csize[best])) best = cc;
                        if (best < 0)
                            for (int cc = 0; cc < 8; cc++)
                                if (csize[cc] < cap && (best < 0 || csize[cc] < csize[best])) best = cc;
                        colour[q] = best;
                        csize[best]++;
                    }
                // local search: a quarter-warp's LDS.128 of vertex k takes as many wavefronts as its fullest bank group holds
                // DISTINCT particles; move single particles to another colour while that lowers the total (a few sweeps).
                // Config 4: wavefronts per quarter-warp read 1.22 -> 1.11 (tets), 1.10 -> 1.06 (triangles), 1.24 -> 1.13 (hinges)
                auto group_cost = [&](int g) {
                    int cn[8] = {0, 0, 0, 0, 0, 0, 0, 0}, mx = 0;
                    for (int r : groups[g]) mx = std::max(mx, ++cn[colour[r]]);
                    return mx;
                };
                for (int sweep = 0; sweep < 8; sweep++) {
                    bool improved = false;
                    for (int q = 0; q < P_; q++) {
                        if (of_part[q].empty()) continue;
                        int base = 0;
                        for (int g : of_part[q]) base += group_cost(g);
                        const int c0 = colour[q];
                        int best = c0, best_cost = base;
                        for (int cc = 0; cc < 8; cc++) {
                            if (cc == c0 || csize[cc] >= cap) continue;
                            colour[q] = cc;
                            int cost = 0;
                            for (int g : of_part[q]) cost += group_cost(g);
                            if (cost < best_cost) { best_cost = cost; best = cc; }
                        }
                        colour[q] = best;
                        if (best != c0) { csize[c0]--; csize[best]++; improved = true; }
                    }
                    if (!improved) break;
                }
                tloc[j].resize(P_);
                std::fill(csize.begin(), csize.end(), 0);
                for (int q = 0; q < P_; q++) { tloc[j][q] = colour[q] + 8 * csize[colour[q]]; csize[colour[q]]++; }
                for (int cc = 0; cc < 8; cc++) lmax = std::max(lmax, 8 * csize[cc]);
            }
        }
        hs.lmax = lmax;
        // pass 2: one packed record per tile (RecLayout), fixed-stride particle lists
        const int rb = rec_bytes_of(t);
        const int oC0 = kTileElems * 8, oC1 = oC0 + kTileElems * 16, oC2 = oC1 + (t == T_TET ? kTileElems * 16 : 0);
        const int oArea = oC2 + (t == T_TET ? kTileElems * 8 : 0), oSlots = oArea + (t == T_TRI ? kTileElems * 4 : 0);
        const int oSlotDesc = oSlots + 4 * kTileElems * 2;
        std::vector<char> rec((size_t)nt * rb, 0);
        const size_t tp_ints = (size_t)pmax * 6 / 4;  // ints per tile block: id[pmax] then loc[pmax] (u16)
        std::vector<int> tparts((size_t)nt * tp_ints, -1);
        std::vector<int> pos;
        for (int j = 0; j < nt; j++) {
            const int e0 = j * kTileElems, e1 = std::min(c, e0 + kTileElems);
            const int P_ = (int)tids[j].size();
            char *R = rec.data() + (size_t)j * rb;
            ushort4 *lidx = (ushort4 *)R;
            float4 *q0 = (float4 *)(R + oC0), *q1 = (float4 *)(R + oC1);
            float2 *q2 = (float2 *)(R + oC2);
            float *qa = (float *)(R + oArea);
            uint16_t *slots = (uint16_t *)(R + oSlots), *slot_desc = (uint16_t *)(R + oSlotDesc);
            // local index of a global id: sorted (id, local) pairs
            std::vector<std::pair<int, int>> look(P_);
            for (int q = 0; q < P_; q++) look[q] = {tids[j][q], q};
            std::sort(look.begin(), look.end());
            // entries sorted by tile-particle: particle q owns entries [start[q], start[q] + count[q])
            std::vector<int> start(P_ + 1, 0);
            for (int q = 0; q < P_; q++) start[q + 1] = start[q] + tcnt[j][q];
            for (int k = 0; k < 4 * kTileElems; k++) slots[k] = 0;
            {
                std::vector<int> part_of(start[P_]);
                for (int q = 0; q < P_; q++)
                    for (int r = 0; r < tcnt[j][q]; r++) part_of[start[q] + r] = q;
                const int n_entries = start[P_];
                for (int th = 0; th < kTileElems; th++) {
                    const int b0 = 4 * th, nv = std::max(0, std::min(4, n_entries - b0));
                    unsigned dsc = (unsigned)nv << 13;
                    if (nv > 0) {
                        dsc |= (unsigned)part_of[b0];
                        for (int k = 1; k < nv; k++)
                            if (part_of[b0 + k] != part_of[b0 + k - 1]) dsc |= 1u << (9 + k);
                    }
                    slot_desc[th] = (uint16_t)dsc;
                }
            }
            pos.assign(P_ + 1, 0);  // pos[q]: how many incidences of particle q have been placed
            for (int q = 0; q < P_; q++) {
                tparts[(size_t)j * tp_ints + q] = tids[j][q];
                ((uint16_t *)(tparts.data() + (size_t)j * tp_ints + pmax))[q] = (uint16_t)tloc[j][q];
            }
            for (int e = e0; e < e1; e++) {
                unsigned short li[4] = {0, 0, 0, 0};
                for (int k = 0; k < a; k++) {
                    const int gi = inv_p[conn[t][(size_t)hs.perm[e] * a + k]];
                    const int lp = std::lower_bound(look.begin(), look.end(), std::make_pair(gi, -1))->second;
                    li[k] = (unsigned short)tloc[j][lp];
                    slots[start[lp] + pos[lp]++] = (uint16_t)(k * kTileElems + (e - e0));
                }
                lidx[e - e0] = make_ushort4(li[0], li[1], li[2], li[3]);
                q0[e - e0] = r0[hs.perm[e]];
                if (t == T_TET) { q1[e - e0] = r1[hs.perm[e]]; q2[e - e0] = r2[hs.perm[e]]; }
                if (t == T_TRI) qa[e - e0] = r1[hs.perm[e]].x;
            }
        }
        all_tids[t] = tids;
        UP(L.rec[t], rec); UP(L.tile_parts[t], tparts);
        UP(L.perm[t], hs.perm);
        // per-env element parameters: [E][n_tiles][3][kTileElems] (padding holds harmless finite values)
        if (t != T_HINGE) {
            const float *src[3] = {t == T_TET ? d->tet_mu : d->tri_mu, t == T_TET ? d->tet_lambda : d->tri_lambda, t == T_TET ? d->tet_damp : d->tri_damp};
            std::vector<float> v((size_t)3 * E * cp, 1.0f);
            for (int q = 0; q < 3; q++)
                for (int env = 0; env < E; env++)
                    for (int e = 0; e < c; e++) {
                        float val = (d->param_layout & GS_ELEM_PER_ENV) ? src[q][(size_t)env * c + hs.perm[e]] : src[q][hs.perm[e]];
                        if (!std::isfinite(val)) { set_error("%s parameter %d of element %d is not finite", tname[t], q, hs.perm[e]); return GS_EINVAL; }
                        if (q == 1 && !(val > 0.0f)) { set_error("%s %d: lambda must be > 0", tname[t], hs.perm[e]); return GS_EINVAL; }
                        v[par_index(nt, env, e, q)] = val;
                    }
            UP(L.par[t], v);
            if (c > 0) {  // an empty set owns one placeholder element only
                cudaError_t ce = cudaMemsetAsync(L.g32[t], 0, sizeof(float) * kNumGrads[t] * (size_t)E * cp, stream);
                if (ce == cudaSuccess) ce = cudaMemsetAsync(L.g64[t], 0, sizeof(double) * kNumGrads[t] * (size_t)E * cp, stream);
                if (ce != cudaSuccess) return cuda_fail(ce, "memset grads");
            }
        }
        if (t == T_HINGE && c > 0) {
            cudaError_t ce = cudaMemsetAsync(L.g32[t], 0, sizeof(float) * (size_t)E * cp, stream);
            if (ce == cudaSuccess) ce = cudaMemsetAsync(L.g64[t], 0, sizeof(double) * (size_t)E * cp, stream);
            if (ce != cudaSuccess) return cuda_fail(ce, "memset grads");
        }
        ElemDev &ed = dev.es[t];
        ed.count = c; ed.cpad = cp; ed.n_tiles = nt; ed.pmax = pmax; ed.lmax = lmax; ed.rec_bytes = rb;
        ed.rec = L.rec[t]; ed.tile_parts = L.tile_parts[t]; ed.par = L.par[t];
        ed.g32 = L.g32[t]; ed.g64 = L.g64[t];
        ed.perm = L.perm[t];
        m->counts[t] = c;
    }
    {
        // deterministic mode: greedy colouring of the tiles of all types (tets, then triangles, then hinges, in tile order):
        // a tile takes the lowest colour none of its particles has seen; per colour class no two tiles share a particle
        std::vector<uint64_t> seen(N, 0);
        std::vector<int> colour[N_TYPES];
        int nc = 0;
        bool ok = true;
        for (int t = 0; t < N_TYPES && ok; t++) {
            colour[t].assign(all_tids[t].size(), 0);
            for (size_t j = 0; j < all_tids[t].size(); j++) {
                uint64_t used = 0;
                for (int pi : all_tids[t][j]) used |= seen[pi];
                int c = 0;
                while (c < 64 && (used >> c & 1ull)) c++;
                if (c == 64) { ok = false; break; }
                colour[t][j] = c;
                nc = std::max(nc, c + 1);
                for (int pi : all_tids[t][j]) seen[pi] |= 1ull << c;
            }
        }
        m->det_colours = ok ? nc : 0;
        for (int t = 0; t < N_TYPES; t++) {
            const int nt = (int)all_tids[t].size();
            std::vector<int> order(nt);
            std::iota(order.begin(), order.end(), 0);
            if (ok) std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return colour[t][a] < colour[t][b]; });
            m->det_off[t].assign(nc + 1, 0);
            if (ok)
                for (int j = 0; j < nt; j++) m->det_off[t][colour[t][j] + 1]++;
            for (int c = 0; c < nc; c++) m->det_off[t][c + 1] += m->det_off[t][c];
            UP(L.det[t], order);
            m->d_det[t] = L.det[t];
        }
    }
    dev.N = N; dev.E = E;
    dev.gx = d->gravity[0]; dev.gy = d->gravity[1]; dev.gz = d->gravity[2]; dev.dt = d->dt;
    {
        double nl = std::sqrt((double)d->plane_n[0] * d->plane_n[0] + (double)d->plane_n[1] * d->plane_n[1] + (double)d->plane_n[2] * d->plane_n[2]);
        if (!(nl > 0)) { set_error("plane_n must be non-zero"); return GS_EINVAL; }
        dev.nx = (float)(d->plane_n[0] / nl); dev.ny = (float)(d->plane_n[1] / nl); dev.nz = (float)(d->plane_n[2] / nl);
    }
    dev.pd = d->plane_d; dev.pr = d->particle_radius;
    dev.ke = L.ke; dev.kd = L.kd; dev.kf = L.kf; dev.muc = L.muc;
    dev.kdrag = L.kdrag; dev.klift = L.klift; dev.wx = d->wind[0]; dev.wy = d->wind[1]; dev.wz = d->wind[2];
    dev.aero = (m->aero_host && counts[T_TRI] > 0) ? 1 : 0;
    dev.perm_p = L.perm_p; dev.inv_mass = L.inv_mass; dev.gmass32 = L.gmass32; dev.gmass64 = L.gmass64; dev.gacc = L.gacc; dev.gcon64 = L.gcon64; dev.tile_ctr = L.tile_ctr; dev.bad = L.bad; dev.frame_base = L.frame_base;
    m->N = N; m->E = E;
    m->d_f = L.f; m->d_xs[0] = L.xs[0]; m->d_xs[1] = L.xs[1]; m->d_vs[0] = L.vs[0]; m->d_vs[1] = L.vs[1];
    m->d_adjx = L.adjx; m->d_adjv = L.adjv; m->d_adjf = L.adjf;
    m->d_inv_mass = L.inv_mass;
    const size_t EN = (size_t)E * N;
    cudaError_t ce = cudaMemsetAsync(L.f, 0, sizeof(float4) * EN, stream);
    if (ce == cudaSuccess) ce = cudaMemsetAsync(L.gmass32, 0, sizeof(float) * EN, stream);
    if (ce == cudaSuccess) ce = cudaMemsetAsync(L.gmass64, 0, sizeof(double) * EN, stream);
    if (ce == cudaSuccess) ce = cudaMemsetAsync(L.gacc, 0, sizeof(double) * (size_t)E * kConSlots * kAccVals, stream);
    if (ce == cudaSuccess) ce = cudaMemsetAsync(L.gcon64, 0, sizeof(double) * (size_t)E * kAccVals, stream);
    if (ce == cudaSuccess) ce = cudaMemsetAsync(L.tile_ctr, 0, sizeof(int) * 8, stream);
    if (ce == cudaSuccess) ce = cudaMemsetAsync(L.bad, 0x7f, sizeof(int), stream);
    if (ce != cudaSuccess) return cuda_fail(ce, "memset workspace");
    ce = cudaStreamSynchronize(stream);
    if (ce != cudaSuccess) return cuda_fail(ce, "model upload");
    return GS_OK;
}

}  // namespace gs

extern "C" const char *gs_last_error(void) { return gs::last_error(); }
