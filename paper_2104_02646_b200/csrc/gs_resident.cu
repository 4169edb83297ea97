// gs_resident.cu -- the RESIDENT plan: one persistent CTA per environment runs ALL substeps of a rollout
// (k_resident_fwd) or of its adjoint (k_resident_adj) in one launch.
//
// For meshes that fit one CTA (BASELINE.json configs[0] and the 1024-environment configs[3]: 125 particles,
// 320 tets) two grid-wide launches per substep are pure launch latency, and streaming the state through HBM
// every substep is wasted traffic.  Here
//   - each thread owns EPT tets for the whole rollout: connectivity, B, V, mu, lambda, k_damp stay in registers;
//   - each particle is served by a group of 1, 2 or 4 adjacent lanes (the largest that fits the CTA); the group's lead
//     lane keeps x, v (forward) or adj_x, adj_v (adjoint) in registers across substeps and mirrors them to shared
//     memory for the element phase;
//   - scatter is a shared-memory gather list: element threads write per-vertex contributions to
//     conflict-free float4 slots, the lanes of a particle's group sum disjoint parts of its slot run and combine
//     them by shuffle -- no atomics, deterministic; particles are assigned to groups in order of valence, so the
//     lanes of a warp run near-equal loops;
//   - the only HBM traffic is the tape: one coalesced float4 store of (x, v) per particle per substep in the
//     forward pass, one prefetched load per substep in the adjoint;
//   - parameter gradients (a10) accumulate in fp32 registers; every 32 substeps the chunk is folded into the fp64
//     masters in global memory (hazard H4; each thread owns its entries, so no atomics).
// Two __syncthreads per substep.  Bound: plain fp32 ALU + barrier latency, not HBM.
//
// Tets only (the element functions are those of gs_elements.cuh, shared with the streaming plan); meshes with
// triangles / hinges, more than kResMaxTets tets or more particles than threads run the streaming plan.
#include <algorithm>
#include <climits>
#include <vector>

#include "gs_elements.cuh"
#include "gs_internal.h"

namespace gs {

constexpr int kResMaxTets = 2048;
constexpr int kResMaxThreads = 1024;

struct ResDev {
    int M, N, nthreads, kpp;   // kpp: lanes per particle in the particle phase (1, 2 or 4)
    int L;                     // size of the shared-memory staging index space (multiple of 8, >= N)
    const ushort4 *idx;        // [M] STAGING indices of each tet's particles (internal element order)
    const uint16_t *rloc;      // [N] staging index of internal particle p: assigned by greedy 8-colouring so that the
                               // particles one quarter-warp reads for the same vertex fall into different 16-byte bank
                               // groups (conflict-free LDS.128), as in the streaming plan
    const uint16_t *owner;     // [N] particle served by particle slot q, most incident tets first
    const uint16_t *csr_ptr;   // [N + 1] incidences per internal particle (prefix sums): valence = ptr[p + 1] - ptr[p]
    // Scatter as a TRANSPOSED gather list.  Particle slots are sorted by valence (most incident tets first), and the j-th
    // incidence of the particle in slot q lives at entry row[j] + q of the contribution plane: row j holds the j-th
    // incidence of every particle that has one (slots 0 .. count_j - 1).  The lanes of a warp serve consecutive slots, so
    // their LDS.128 of one row are consecutive, conflict-free, and need no index load; with kpp lanes per particle the lanes
    // of a group take rows j0, j0 + kpp, ..., and row starts are padded to 8 / kpp modulo 8 entries so that the rows a
    // quarter-warp reads at once fall into different 16-byte bank groups.  Element threads keep the four destinations of
    // their tet in two registers.
    const ushort4 *dest;       // [M] entry of each tet vertex's contribution
    const uint16_t *row;       // [maxval + 1] first entry of row j
    int maxval, Ltot;          // rows; entries of one contribution plane (padded)
};

// activation schedule of the tets (gs_actuation_create), internal order [F][E][cpad]; used by the ACT kernel variants
struct ResAct {
    const float *tet;
    float *g_tet;
    int F, stride;
    size_t fstride;  // E * cpad
};

// The forward and the adjoint kernel may use different layouts of the particle phase (the tape is indexed by particle, so the
// two need not agree): the lean forward kernel runs best with two tets per thread and half the threads where the particles
// still fit, the adjoint with one tet per thread.  rd_fwd shares idx / rloc / csr_ptr with rd; owner / dest / row are its own.
struct ResHost {
    ResDev rd, rd_fwd;
    int ept, ept_fwd;
    size_t smem_fwd, smem_adj;
};

static inline size_t al16(size_t n) { return (n + 15) & ~(size_t)15; }

// shared memory: sx[N] float4, sv[N] float4, (adjoint: sa[N] float4), contributions [planes][Ltot] float4, csr_ptr, owner, row
// adjoint only: per-particle accumulators of the per-environment totals (contact parameters, gravity): double[7][N] masters,
// then float[7][N] chunks
constexpr int kResAcc = 7;
static size_t res_smem(int L, int N, int Ltot, int maxval, int planes, bool adj) {
    return (size_t)(adj ? 3 : 2) * L * sizeof(float4) + (size_t)planes * Ltot * sizeof(float4) + (adj ? al16((size_t)N * (kResAcc * 8 + kResAcc * 4)) : 0) +
           al16((size_t)(N + 1) * 2) + al16((size_t)N * 2) + al16((size_t)(maxval + 1) * 2);
}
static int res_ept(int M) { return M > kResMaxThreads ? 2 : 1; }
// forward: two tets per thread where half the threads still hold one particle each AND the batch fills the GPU (more than two
// CTAs per SM: throughput-bound).  A small batch is latency-bound per CTA and runs faster with one tet per thread
// (config 0, one environment: forward 2.6 ms against 3.2 ms).
constexpr int kResBatchEnvs = 2 * 148;
static int res_ept_fwd(int M, int N, int E) {
    return (M > kResMaxThreads || (E > kResBatchEnvs && ((M + 1) / 2 + 31) / 32 * 32 >= N)) ? 2 : 1;
}
static int res_threads(int M, int ept) { return ((M + ept - 1) / ept + 31) / 32 * 32; }
static int res_kpp(int nthreads, int N) { return nthreads >= 4 * N ? 4 : (nthreads >= 2 * N ? 2 : 1); }
// rows of the transposed gather list from the valences (any order): row[j] (maxval + 1 entries); returns the padded total.
// Row starts are placed at prescribed residues modulo 8 (the 16-byte bank group of entry row[j] + q is (row[j] + q) mod 8):
// the rows a lane group reads in the same iteration (kpp = 2: rows 2i, 2i + 1; kpp = 4: rows 4i .. 4i + 3) must differ by
// 8 / kpp so that a quarter-warp's LDS.128 is conflict-free, and beyond that the residues cycle through all eight values,
// which gives the store side (res_dest) up to eight bank groups to choose from for every incidence of a particle.
static int res_rows(std::vector<int> val, int kpp, std::vector<uint16_t> *row) {
    static const int kRes2[8] = {0, 4, 1, 5, 2, 6, 3, 7}, kRes4[8] = {0, 2, 4, 6, 1, 3, 5, 7};
    std::sort(val.begin(), val.end(), [](int a, int b) { return a > b; });
    const int maxval = val.empty() ? 0 : val[0];
    int off = 0;
    if (row) row->assign(maxval + 1, 0);
    for (int j = 0; j < maxval; j++) {
        const int want = kpp == 2 ? kRes2[j & 7] : (kpp == 4 ? kRes4[j & 7] : (j & 7));
        while ((off & 7) != want) off++;
        int cnt = 0;
        while (cnt < (int)val.size() && val[cnt] > j) cnt++;
        if (row) (*row)[j] = (uint16_t)off;
        off += cnt;
    }
    if (row) (*row)[maxval] = (uint16_t)off;
    return off;
}
static std::vector<int> res_valences(const gs_model_desc *d) {
    std::vector<int> val(d->n_particles, 0);
    for (size_t i = 0; i < (size_t)d->n_tets * 4; i++) {
        const int p = d->tets[i];
        if (p >= 0 && p < d->n_particles) val[p]++;
    }
    return val;
}

static bool resident_fits(const gs_model_desc *d) {
    if (d->n_tris > 0 || d->n_hinges > 0 || d->n_tets < 1 || d->n_tets > kResMaxTets) return false;
    const int nthreads = res_threads(d->n_tets, res_ept(d->n_tets));
    if (d->n_particles > nthreads || !d->tets) return false;
    const std::vector<int> val = res_valences(d);
    const int maxval = *std::max_element(val.begin(), val.end());
    const int Ltot = res_rows(val, res_kpp(nthreads, d->n_particles), nullptr);
    const int nthreads_f = res_threads(d->n_tets, res_ept_fwd(d->n_tets, d->n_particles, d->n_envs));
    const int Ltot_f = res_rows(val, res_kpp(nthreads_f, d->n_particles), nullptr);
    if (Ltot > 65535 || Ltot_f > 65535) return false;
    return res_smem(d->n_particles + 24, d->n_particles, Ltot, maxval, 2, true) <= 200 * 1024 &&
           res_smem(d->n_particles + 24, d->n_particles, Ltot_f, maxval, 1, false) <= 200 * 1024;
}

size_t resident_blob_bytes(const gs_model_desc *d) {
    if (!resident_fits(d)) return 0;
    // idx, csr_ptr, rloc once; dest, row, owner per layout (adjoint, forward)
    return 256 * 12 + 3 * (size_t)d->n_tets * sizeof(ushort4) + (size_t)(4 * d->n_particles + 1) * 2 + 2 * (size_t)(4 * d->n_tets + 2) * 2;
}

// ------------------------------------------------------------------------------------------ kernels
struct TetReg {
    float b[9], V, mu, lam, kd;
    float act;  // this substep's actuation; 0 in the passive kernels
    ushort4 li;   // staging indices of the four particles
    ushort4 dst;  // entries of the four per-vertex contributions (ResDev::dest)
    bool on;
};

template <int EPT>
__device__ __forceinline__ void load_tets(const ModelDev &md, const ResDev &rd, int env, TetReg tr[EPT]) {
    const ElemDev &es = md.es[T_TET];
#pragma unroll
    for (int j = 0; j < EPT; j++) {
        const int e = threadIdx.x + j * blockDim.x;
        tr[j].on = e < rd.M;
        const int ee = tr[j].on ? e : 0;
        using R = RecLayout<T_TET>;
        const char *rec = es.rec + (size_t)(ee / kTileElems) * es.rec_bytes;
        const int el = ee % kTileElems;
        const float4 c0 = ((const float4 *)(rec + R::oC0))[el], c1 = ((const float4 *)(rec + R::oC1))[el];
        const float2 c2 = ((const float2 *)(rec + R::oC2))[el];
        tr[j].b[0] = c0.x; tr[j].b[1] = c0.y; tr[j].b[2] = c0.z; tr[j].b[3] = c0.w;
        tr[j].b[4] = c1.x; tr[j].b[5] = c1.y; tr[j].b[6] = c1.z; tr[j].b[7] = c1.w; tr[j].b[8] = c2.x;
        tr[j].V = c2.y;
        tr[j].mu = es.par[par_index(es.n_tiles, env, ee, 0)];
        tr[j].lam = es.par[par_index(es.n_tiles, env, ee, 1)];
        tr[j].kd = es.par[par_index(es.n_tiles, env, ee, 2)];
        tr[j].li = rd.idx[ee];
        tr[j].dst = rd.dest[ee];
        tr[j].act = 0.0f;
    }
}

__device__ __forceinline__ void load_csr(const ResDev &rd, uint16_t *s_ptr, uint16_t *s_owner, uint16_t *s_row) {
    for (int i = threadIdx.x; i <= rd.N; i += blockDim.x) s_ptr[i] = rd.csr_ptr[i];
    for (int i = threadIdx.x; i < rd.N; i += blockDim.x) s_owner[i] = rd.owner[i];
    for (int i = threadIdx.x; i <= rd.maxval; i += blockDim.x) s_row[i] = rd.row[i];
}

// Particle ownership: particle slot q = tid / kpp is served by kpp adjacent lanes (kpp = 1, 2 or 4, the largest that
// fits the CTA); slot q owns particle owner[q] (particles sorted by valence, so the lanes of a warp have near-equal
// trip counts).  Lane j of the group sums the j-th part of the particle's slot run; the parts meet by shuffle and
// lane 0 (the "lead") holds the particle's state in registers for the whole rollout.
struct PartOwn {
    bool is_p, lead;
    int p, lp;          // particle, its staging index
    int q, j0, val;     // particle slot; this lane takes rows j0, j0 + kpp, ... < val of the particle's incidences
};
__device__ __forceinline__ PartOwn part_own(const ResDev &rd, const uint16_t *s_ptr, const uint16_t *s_owner) {
    PartOwn o;
    const int q = threadIdx.x / rd.kpp, j = threadIdx.x % rd.kpp;
    o.is_p = q < rd.N;
    o.lead = o.is_p && j == 0;
    o.p = o.is_p ? s_owner[q] : 0;
    o.lp = rd.rloc[o.p];
    o.q = q; o.j0 = j;
    o.val = o.is_p ? s_ptr[o.p + 1] - s_ptr[o.p] : 0;
    return o;
}
__device__ __forceinline__ float group_sum(float v, int kpp) {
    if (kpp >= 2) v += __shfl_xor_sync(0xffffffffu, v, 1);
    if (kpp >= 4) v += __shfl_xor_sync(0xffffffffu, v, 2);
    return v;
}

// forward: substeps [0, T), tape slot s = (x4, v4) at base + 2 s S (+ S for v), S = E N
template <int EPT, int MAXT, int MINB, bool ACT>
__global__ void __launch_bounds__(MAXT, MINB) k_resident_fwd(const ModelDev md, const ResDev rd, float4 *__restrict__ tape, size_t S, int T, const ResAct ra) {
    extern __shared__ float4 smem4[];
    const int N = rd.N, M = rd.M, L = rd.L;
    float4 *sx = smem4, *sv = smem4 + L;
    float4 *sf = smem4 + 2 * L;  // [Ltot] per element-vertex force, transposed gather layout
    uint16_t *s_ptr = reinterpret_cast<uint16_t *>(sf + rd.Ltot);
    uint16_t *s_owner = s_ptr + (((N + 1) + 7) & ~7);
    uint16_t *s_row = s_owner + ((N + 7) & ~7);
    const int tid = threadIdx.x, env = blockIdx.x;
    TetReg tr[EPT];
    load_tets<EPT>(md, rd, env, tr);
    load_csr(rd, s_ptr, s_owner, s_row);
    __syncthreads();
    const PartOwn po = part_own(rd, s_ptr, s_owner);
    const size_t poff = (size_t)env * N + po.p;
    float4 xq = make_float4(0.f, 0.f, 0.f, 0.f), vq = xq;
    if (po.lead) { xq = tape[poff]; vq = tape[S + poff]; sx[po.lp] = xq; sv[po.lp] = vq; }
    ContactParams cp;
    cp.n = vec3(md.nx, md.ny, md.nz); cp.d = md.pd; cp.r = md.pr;
    cp.ke = md.ke[env]; cp.kd = md.kd[env]; cp.kf = md.kf[env]; cp.mu = md.muc[env];
    const vec3 g(md.gx, md.gy, md.gz);
    __syncthreads();
    int bad = INT_MAX;
    float4 *tpf = tape + poff;  // this particle's entry of the current tape slot (x; v is S further)
    for (int s = 0; s < T; s++) {
        if (ACT && s % ra.stride == 0 && s / ra.stride < ra.F) {  // a new frame of the activation schedule begins
#pragma unroll
            for (int j = 0; j < EPT; j++)
                if (tr[j].on) tr[j].act = ra.tet[(size_t)(s / ra.stride) * ra.fstride + (size_t)env * md.es[T_TET].cpad + tid + j * blockDim.x];
        }
#pragma unroll
        for (int j = 0; j < EPT; j++) {
            if (tr[j].on) {
                const ushort4 li = tr[j].li;
                const vec3 x[4] = {vec3(sx[li.x]), vec3(sx[li.y]), vec3(sx[li.z]), vec3(sx[li.w])};
                const vec3 v[4] = {vec3(sv[li.x]), vec3(sv[li.y]), vec3(sv[li.z]), vec3(sv[li.w])};
                vec3 f[4];
                tet_force(x, v, tr[j].b, tr[j].V, tr[j].mu, tr[j].lam, tr[j].kd, tr[j].act, f);
                const ushort4 ds = tr[j].dst;
                sf[ds.x] = make_float4(f[0].x, f[0].y, f[0].z, 0.f); sf[ds.y] = make_float4(f[1].x, f[1].y, f[1].z, 0.f);
                sf[ds.z] = make_float4(f[2].x, f[2].y, f[2].z, 0.f); sf[ds.w] = make_float4(f[3].x, f[3].y, f[3].z, 0.f);
            }
        }
        __syncthreads();
        float ax = 0.f, ay = 0.f, az = 0.f;
        for (int j = po.j0; j < po.val; j += rd.kpp) {
            const float4 c = sf[s_row[j] + po.q];
            ax += c.x; ay += c.y; az += c.z;
        }
        ax = group_sum(ax, rd.kpp); ay = group_sum(ay, rd.kpp); az = group_sum(az, rd.kpp);
        if (po.lead) {
            const vec3 x(xq), v(vq);
            const vec3 f = vec3(ax, ay, az) + contact_force(cp, x, v);
            vec3 x1, v1;
            integrate(x, v, f, xq.w, g, md.dt, x1, v1);
            xq = make_float4(x1.x, x1.y, x1.z, xq.w);
            vq = make_float4(v1.x, v1.y, v1.z, 0.f);
            sx[po.lp] = xq; sv[po.lp] = vq;
            tpf += 2 * S;
            tpf[0] = xq; tpf[S] = vq;
            const float chk = x1.x + x1.y + x1.z + v1.x + v1.y + v1.z;
            if (!(fabsf(chk) <= 3.0e38f) && bad == INT_MAX) bad = s;
        }
        __syncthreads();
    }
    if (bad != INT_MAX) atomicMin(md.bad, bad);
}

// adjoint: substeps T-1 .. 0.  adjx / adjv: [E][N] float4 in/out (dL/d(final state) -> dL/d(initial state)).
// frames: caller-order [n_frames][E][N][3] cotangents of the states after (k+1) * stride substeps, or nullptr.
template <int EPT, int MAXT, int MINB, bool ACT>
__global__ void __launch_bounds__(MAXT, MINB) k_resident_adj(const ModelDev md, const ResDev rd, const float4 *__restrict__ tape, size_t S, int T,
                                                              float4 *__restrict__ adjx, float4 *__restrict__ adjv, const float *__restrict__ frames,
                                                              int n_frames, int stride, const ResAct ra) {
    extern __shared__ float4 smem4[];
    const int N = rd.N, PL = rd.Ltot, L = rd.L;
    float4 *sx = smem4, *sv = smem4 + L, *sa = smem4 + 2 * L;
    float4 *sf = smem4 + 3 * L;  // [2][Ltot]: adj_x contributions, then adj_v contributions, per element-vertex (transposed gather layout)
    // dL/d(k_e, k_d, k_f, mu_c) and dL/dg: per-particle partial sums (only the particle's lead lane touches its entries):
    // fp32 chunks of kFlushEvery substeps in shared memory (no registers held across the element phase) folded into fp64
    // masters (hazard H4), summed in particle order at the end: deterministic
    double *dgc = reinterpret_cast<double *>(sf + 2 * PL);   // [kResAcc][N]
    float *sgc = reinterpret_cast<float *>(dgc + kResAcc * N);  // [kResAcc][N]
    uint16_t *s_ptr = reinterpret_cast<uint16_t *>(reinterpret_cast<char *>(dgc) + ((N * (kResAcc * 8 + kResAcc * 4) + 15) & ~15));
    uint16_t *s_owner = s_ptr + (((N + 1) + 7) & ~7);
    uint16_t *s_row = s_owner + ((N + 7) & ~7);
    const int tid = threadIdx.x, env = blockIdx.x;
    TetReg tr[EPT];
    load_tets<EPT>(md, rd, env, tr);
    load_csr(rd, s_ptr, s_owner, s_row);
    __syncthreads();
    const PartOwn po = part_own(rd, s_ptr, s_owner);
    const size_t poff = (size_t)env * N + po.p;
    ContactParams cp;
    cp.n = vec3(md.nx, md.ny, md.nz); cp.d = md.pd; cp.r = md.pr;
    cp.ke = md.ke[env]; cp.kd = md.kd[env]; cp.kf = md.kf[env]; cp.mu = md.muc[env];
    const vec3 g(md.gx, md.gy, md.gz);
    const float dt = md.dt;
    vec3 bx = zero3(), bv = zero3();       // running cotangents of the lead thread's particle
    float4 xq = make_float4(0.f, 0.f, 0.f, 0.f), vq = xq, vnext = xq;
    const float *cot = nullptr;
    if (po.lead) {
        bx = vec3(adjx[poff]); bv = vec3(adjv[poff]);
        vnext = tape[(size_t)(2 * T + 1) * S + poff];
        xq = tape[(size_t)(2 * (T - 1)) * S + poff]; vq = tape[(size_t)(2 * (T - 1) + 1) * S + poff];
        if (frames) cot = frames + ((size_t)env * N + md.perm_p[po.p]) * 3;
    }
    if (po.lead)
        for (int q = 0; q < kResAcc; q++) { dgc[q * N + po.p] = 0.0; sgc[q * N + po.p] = 0.f; }
    const size_t frame_elems = (size_t)md.E * N * 3;
    const size_t gstride = (size_t)md.E * md.es[T_TET].cpad;
    float gm32 = 0.f;
    float g32[EPT][3];
#pragma unroll
    for (int j = 0; j < EPT; j++)
#pragma unroll
        for (int q = 0; q < 3; q++) g32[j][q] = 0.f;
    // the summed element contributions of the previous element phase, for this thread's particle (lead lane holds them)
    auto gather = [&](vec3 &dx, vec3 &dv) {
        float ax = 0.f, ay = 0.f, az = 0.f, cx = 0.f, cy = 0.f, cz = 0.f;
        for (int j = po.j0; j < po.val; j += rd.kpp) {
            const int sl = s_row[j] + po.q;
            const float4 c = sf[sl], d = sf[PL + sl];
            ax += c.x; ay += c.y; az += c.z;
            cx += d.x; cy += d.y; cz += d.z;
        }
        dx = vec3(group_sum(ax, rd.kpp), group_sum(ay, rd.kpp), group_sum(az, rd.kpp));
        dv = vec3(group_sum(cx, rd.kpp), group_sum(cy, rd.kpp), group_sum(cz, rd.kpp));
    };
    float gact[EPT];
#pragma unroll
    for (int j = 0; j < EPT; j++) gact[j] = 0.f;
    int act_frame = -1;
    // running pointers / counters instead of per-substep 64-bit index products and divisions by the frame stride
    const float4 *tp = tape + (size_t)(2 * (T - 1)) * S + poff;  // state slot of substep s - 1 is tp - 2 S
    const size_t S2 = 2 * S;
    // frame boundary bookkeeping: the state after substep s is frame (s + 1) / stride - 1 when stride divides s + 1
    int fr_left = (T % stride);              // substeps until the next (lower) frame boundary: 0 = state T is one
    int fr_idx = T / stride - 1;             // index of that frame
    for (int s = T - 1; s >= 0; s--) {
        if (ACT) {  // the frame of the activation schedule that holds during substep s
            const int f = s / ra.stride < ra.F ? s / ra.stride : ra.F - 1;
            if (f != act_frame) {
                act_frame = f;
#pragma unroll
                for (int j = 0; j < EPT; j++)
                    if (tr[j].on) tr[j].act = ra.tet[(size_t)f * ra.fstride + (size_t)env * md.es[T_TET].cpad + tid + j * blockDim.x];
            }
        }
        // prefetch the start state of the previous substep while this one is processed
        float4 xp = xq, vp = vq;
        tp -= S2;
        if (po.lead && s > 0) { xp = tp[0]; vp = tp[S]; }
        if (s != T - 1) {  // contributions of the element phase of substep s + 1 (all lanes: the sums meet by shuffle)
            vec3 dx, dv;
            gather(dx, dv);
            bx += dx; bv += dv;
        }
        if (po.lead) {
            if (cot && fr_left == 0 && fr_idx < n_frames) {
                const float *c = cot + (size_t)fr_idx * frame_elems;
                bx += vec3(c[0], c[1], c[2]);
            }
            const float w = xq.w;
            const vec3 x(xq), v(vq);
            const vec3 lv = madd(bv, dt, bx);
            const vec3 af = (dt * w) * lv;
            vec3 ax = bx, av = lv;
            if (w > 0.0f) {
                const vec3 dvf = (vec3(vnext) - v) - dt * g;
                gm32 += -w * dot(dvf, lv);
                if (md.want_gravity) {  // dL/dg = dt sum lv over the free particles
                    sgc[4 * N + po.p] += dt * lv.x; sgc[5 * N + po.p] += dt * lv.y; sgc[6 * N + po.p] += dt * lv.z;
                }
            }
            float gp[4];
            contact_adjoint(cp, x, v, af, ax, av, gp);
            if (gp[0] != 0.f || gp[1] != 0.f || gp[2] != 0.f || gp[3] != 0.f) {
#pragma unroll
                for (int q = 0; q < 4; q++) sgc[q * N + po.p] += gp[q];
            }
            bx = ax; bv = av;
            sx[po.lp] = xq; sv[po.lp] = vq; sa[po.lp] = make_float4(af.x, af.y, af.z, 0.f);
            vnext = vq; xq = xp; vq = vp;
        }
        __syncthreads();
#pragma unroll
        for (int j = 0; j < EPT; j++) {
            if (tr[j].on) {
                const ushort4 li = tr[j].li;
                const vec3 x[4] = {vec3(sx[li.x]), vec3(sx[li.y]), vec3(sx[li.z]), vec3(sx[li.w])};
                const vec3 v[4] = {vec3(sv[li.x]), vec3(sv[li.y]), vec3(sv[li.z]), vec3(sv[li.w])};
                const vec3 a[4] = {vec3(sa[li.x]), vec3(sa[li.y]), vec3(sa[li.z]), vec3(sa[li.w])};
                vec3 ax[4], av[4];
                float gmu, glam, gk, ga;
                tet_adjoint(x, v, a, tr[j].b, tr[j].V, tr[j].mu, tr[j].lam, tr[j].kd, tr[j].act, ax, av, gmu, glam, gk, ga);
                g32[j][0] += gmu; g32[j][1] += glam; g32[j][2] += gk;
                if (ACT) gact[j] += ga;
                const ushort4 ds = tr[j].dst;
                const unsigned dk[4] = {ds.x, ds.y, ds.z, ds.w};
#pragma unroll
                for (int k = 0; k < 4; k++) {
                    sf[dk[k]] = make_float4(ax[k].x, ax[k].y, ax[k].z, 0.f);
                    sf[PL + dk[k]] = make_float4(av[k].x, av[k].y, av[k].z, 0.f);
                }
            }
        }
        if (ACT && s % ra.stride == 0 && s / ra.stride < ra.F) {  // substep s was the first of its frame: the frame's gradient is complete
#pragma unroll
            for (int j = 0; j < EPT; j++) {
                if (tr[j].on) ra.g_tet[(size_t)act_frame * ra.fstride + (size_t)env * md.es[T_TET].cpad + tid + j * blockDim.x] += gact[j];
                gact[j] = 0.f;
            }
        }
        if (fr_left == 0) { fr_left = stride; fr_idx--; }
        fr_left--;
        if ((s & (kFlushEvery - 1)) == 0) {  // fold the fp32 chunk into fp64 (hazard H4)
            if (po.lead) {
#pragma unroll
                for (int q = 0; q < kResAcc; q++) { dgc[q * N + po.p] += (double)sgc[q * N + po.p]; sgc[q * N + po.p] = 0.f; }
            }
            // the fp64 masters live in global memory (each thread owns its entries; one update per kFlushEvery substeps),
            // which keeps 8 registers free for the element VJP
            if (po.lead) md.gmass64[poff] += (double)gm32;
            gm32 = 0.f;
#pragma unroll
            for (int j = 0; j < EPT; j++)
#pragma unroll
                for (int q = 0; q < 3; q++) {
                    if (tr[j].on) md.es[T_TET].g64[q * gstride + (size_t)env * md.es[T_TET].cpad + tid + j * blockDim.x] += (double)g32[j][q];
                    g32[j][q] = 0.f;
                }
        }
        __syncthreads();
    }
    {
        vec3 dx, dv;
        gather(dx, dv);
        bx += dx; bv += dv;
    }
    if (po.lead) {
        adjx[poff] = make_float4(bx.x, bx.y, bx.z, 0.f);
        adjv[poff] = make_float4(bv.x, bv.y, bv.z, 0.f);
    }
    __syncthreads();
    if (tid < kResAcc) {
        double t = 0.0;
        for (int p = 0; p < N; p++) t += dgc[tid * N + p];
        md.gcon64[(size_t)env * kAccVals + tid] += t;
    }
}

// ------------------------------------------------------------------------------------------ host
#define GS_RES_CHECK(what)                                           \
    do {                                                             \
        cudaError_t e_ = cudaGetLastError();                         \
        if (e_ != cudaSuccess) return cuda_fail(e_, what);           \
        count_launch();                                              \
    } while (0)

static ResHost *res_of(gs_model *m) { return (ResHost *)m->res_host; }

template <class K>
static int set_smem(K kern, size_t bytes) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    return e == cudaSuccess ? GS_OK : cuda_fail(e, "cudaFuncSetAttribute (resident)");
}

int resident_prepare(gs_model *m, const gs_model_desc *d, void *d_workspace, size_t bytes, cudaStream_t st) {
    const bool fits = resident_fits(d);
    if (d->plan == GS_PLAN_RESIDENT && !fits) {
        set_error("the resident plan needs a tets-only mesh with <= %d tets and no more particles than threads", kResMaxTets);
        return GS_EINVAL;
    }
    if (d->plan == GS_PLAN_STREAMING || !fits) { m->plan = GS_PLAN_STREAMING; return GS_OK; }
    const int N = d->n_particles, M = d->n_tets;
    const int counts[N_TYPES] = {d->n_tets, d->n_tris, d->n_hinges};
    const size_t off = workspace_bytes_upper(N, d->n_envs, counts);
    if (off + resident_blob_bytes(d) > bytes) { set_error("workspace too small for the resident plan"); return GS_EINVAL; }
    std::vector<int> inv_p(N);
    for (int i = 0; i < N; i++) inv_p[m->perm_p[i]] = i;
    std::vector<ushort4> idx(M);
    std::vector<uint16_t> ptr(N + 1, 0);
    std::vector<int> cnt(N + 1, 0);
    for (int e = 0; e < M; e++) {
        const int32_t *ix = d->tets + (size_t)m->hes[T_TET].perm[e] * 4;
        const int li[4] = {inv_p[ix[0]], inv_p[ix[1]], inv_p[ix[2]], inv_p[ix[3]]};
        idx[e] = make_ushort4((unsigned short)li[0], (unsigned short)li[1], (unsigned short)li[2], (unsigned short)li[3]);
        for (int k = 0; k < 4; k++) cnt[li[k] + 1]++;
    }
    for (int p = 0; p < N; p++) cnt[p + 1] += cnt[p];
    for (int p = 0; p <= N; p++) ptr[p] = (uint16_t)cnt[p];
    const std::vector<ushort4> pid = idx;  // internal particle ids of every tet (idx becomes staging indices below)
    // staging indices by greedy 8-colouring of the (quarter-warp, vertex) read groups
    std::vector<uint16_t> rloc(N);
    int Lsp = 8;
    {
        const int nq = (M + 7) / 8;
        std::vector<std::vector<int>> groups((size_t)nq * 4), of_part(N);
        for (int e = 0; e < M; e++) {
            const int li[4] = {idx[e].x, idx[e].y, idx[e].z, idx[e].w};
            for (int k = 0; k < 4; k++) {
                const int g = (e / 8) * 4 + k;
                if (std::find(groups[g].begin(), groups[g].end(), li[k]) == groups[g].end()) { groups[g].push_back(li[k]); of_part[li[k]].push_back(g); }
            }
        }
        std::vector<int> colour(N, -1), csize(8, 0);
        const int cap = (N + 7) / 8 + 1;
        auto assign = [&](int q) {
            if (colour[q] >= 0) return;
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
        };
        for (int e = 0; e < M; e++) { assign(idx[e].x); assign(idx[e].y); assign(idx[e].z); assign(idx[e].w); }
        for (int q = 0; q < N; q++) assign(q);  // particles no tet touches
        // local search: a quarter-warp's LDS.128 of vertex k takes as many wavefronts as its fullest bank group holds
        // DISTINCT particles; move single particles to another colour while that lowers the total (a few sweeps)
        auto group_cost = [&](int g) {
            int cnt[8] = {0, 0, 0, 0, 0, 0, 0, 0}, mx = 0;
            for (int r : groups[g]) mx = std::max(mx, ++cnt[colour[r]]);
            return mx;
        };
        for (int sweep = 0; sweep < 8; sweep++) {
            bool improved = false;
            for (int q = 0; q < N; q++) {
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
        std::fill(csize.begin(), csize.end(), 0);
        for (int q = 0; q < N; q++) { rloc[q] = (uint16_t)(colour[q] + 8 * csize[colour[q]]); csize[colour[q]]++; }
        for (int cc = 0; cc < 8; cc++) Lsp = std::max(Lsp, 8 * csize[cc]);
        for (int e = 0; e < M; e++) idx[e] = make_ushort4(rloc[idx[e].x], rloc[idx[e].y], rloc[idx[e].z], rloc[idx[e].w]);
    }
    char *p = (char *)d_workspace + off;
    auto take = [&](size_t n) { char *q = p; p += (n + 255) & ~(size_t)255; return q; };
    ushort4 *d_idx = (ushort4 *)take(idx.size() * sizeof(ushort4));
    uint16_t *d_ptr = (uint16_t *)take(ptr.size() * 2);

    // One layout of the particle phase and of the transposed gather list for a CTA of nthreads_ threads (owner / row / dest
    // depend on the lanes per particle); uploaded into the workspace, pointers and sizes into rd.
    cudaError_t ce = cudaSuccess;
    uint16_t *d_rloc = (uint16_t *)take(rloc.size() * 2);
    auto build_layout = [&](int nthreads_, ResDev &rd) {
        // particle slots: most incident tets first (stable), so the lanes of a warp run near-equal gather loops
        std::vector<uint16_t> owner(N);
        for (int i = 0; i < N; i++) owner[i] = (uint16_t)i;
        std::stable_sort(owner.begin(), owner.end(), [&](uint16_t x, uint16_t y) { return cnt[x + 1] - cnt[x] > cnt[y + 1] - cnt[y]; });
        const int kpp_ = res_kpp(nthreads_, N);
        {
            // within a class of equal valence the order is free: arrange it so that the lead lanes of a quarter-warp (8 / kpp
            // particle slots) own particles in different 16-byte bank groups of the staging arrays -- their STS.128 of x, v
            // (and adj_f) after the particle phase are then conflict-free where the class is large enough
            const int per = 8 / kpp_;
            for (int a = 0; a < N;) {
                int b = a;
                const int va = cnt[owner[a] + 1] - cnt[owner[a]];
                while (b < N && cnt[owner[b] + 1] - cnt[owner[b]] == va) b++;
                for (int i = a; i < b; i++) {
                    unsigned banks = 0;
                    for (int j = i - i % per; j < i; j++) banks |= 1u << (rloc[owner[j]] & 7);
                    for (int j = i; j < b; j++)
                        if (!(banks >> (rloc[owner[j]] & 7) & 1u)) { std::swap(owner[i], owner[j]); break; }
                }
                a = b;
            }
        }
        // transposed gather list (ResDev::dest / row): the j-th incidence (element order) of the particle in slot q -> row[j] + q
        std::vector<int> val(N);
        for (int i = 0; i < N; i++) val[i] = cnt[i + 1] - cnt[i];
        std::vector<uint16_t> row;
        const int Ltot = res_rows(val, kpp_, &row);
        const int maxval = (int)row.size() - 1;
        std::vector<int> slot_of(N);
        for (int q = 0; q < N; q++) slot_of[owner[q]] = q;
        // Which of a particle's rows an incidence takes is free: pick it so that the eight lanes of a quarter-warp (eight
        // consecutive tets, same vertex position) store into different 16-byte bank groups where possible (STS.128 is served
        // a quarter-warp at a time); greedy, lowest free row first among the rows whose bank group is still unused.
        std::vector<std::vector<char>> used(N);
        for (int i = 0; i < N; i++) used[i].assign(val[i], 0);
        std::vector<ushort4> dest(M);
        for (int e0 = 0; e0 < M; e0 += 8) {
            for (int k = 0; k < 4; k++) {
                unsigned banks = 0;
                for (int e = e0; e < std::min(M, e0 + 8); e++) {
                    const int pk = k == 0 ? pid[e].x : (k == 1 ? pid[e].y : (k == 2 ? pid[e].z : pid[e].w));
                    int pick = -1, fallback = -1;
                    for (int j = 0; j < val[pk]; j++) {
                        if (used[pk][j]) continue;
                        if (fallback < 0) fallback = j;
                        if (!(banks >> ((row[j] + slot_of[pk]) & 7) & 1u)) { pick = j; break; }
                    }
                    if (pick < 0) pick = fallback;
                    used[pk][pick] = 1;
                    const unsigned short dk = (unsigned short)(row[pick] + slot_of[pk]);
                    banks |= 1u << (dk & 7);
                    if (k == 0) dest[e].x = dk; else if (k == 1) dest[e].y = dk; else if (k == 2) dest[e].z = dk; else dest[e].w = dk;
                }
            }
        }
        {
            // local search on the store side: a quarter-warp's STS.128 of vertex k takes as many wavefronts as its fullest
            // bank group holds entries; swap the rows of two incidences of one particle while that lowers the total
            auto dk = [&](int e, int k) -> unsigned short & { return k == 0 ? dest[e].x : (k == 1 ? dest[e].y : (k == 2 ? dest[e].z : dest[e].w)); };
            auto grp_cost = [&](int e, int k) {
                int cnt[8] = {0, 0, 0, 0, 0, 0, 0, 0}, mx = 0;
                const int e0 = e & ~7;
                for (int f = e0; f < std::min(M, e0 + 8); f++) mx = std::max(mx, ++cnt[dk(f, k) & 7]);
                return mx;
            };
            std::vector<std::vector<std::pair<int, int>>> inc(N);
            for (int e = 0; e < M; e++) {
                const unsigned short pk[4] = {pid[e].x, pid[e].y, pid[e].z, pid[e].w};
                for (int k = 0; k < 4; k++) inc[pk[k]].push_back({e, k});
            }
            for (int sweep = 0; sweep < 8; sweep++) {
                bool improved = false;
                for (int q = 0; q < N; q++)
                    for (size_t a = 0; a < inc[q].size(); a++)
                        for (size_t b = a + 1; b < inc[q].size(); b++) {
                            const int ea = inc[q][a].first, ka = inc[q][a].second, eb = inc[q][b].first, kb = inc[q][b].second;
                            if ((ea & ~7) == (eb & ~7) && ka == kb) continue;  // same store instruction of the same quarter-warp
                            const int before = grp_cost(ea, ka) + grp_cost(eb, kb);
                            std::swap(dk(ea, ka), dk(eb, kb));
                            if (grp_cost(ea, ka) + grp_cost(eb, kb) < before) improved = true;
                            else std::swap(dk(ea, ka), dk(eb, kb));
                        }
                if (!improved) break;
            }
        }
        ushort4 *d_dest = (ushort4 *)take(dest.size() * sizeof(ushort4));
        uint16_t *d_row = (uint16_t *)take(row.size() * 2);
        uint16_t *d_owner = (uint16_t *)take(owner.size() * 2);
        if (ce == cudaSuccess) ce = cudaMemcpyAsync(d_owner, owner.data(), owner.size() * 2, cudaMemcpyHostToDevice, st);
        if (ce == cudaSuccess) ce = cudaMemcpyAsync(d_dest, dest.data(), dest.size() * sizeof(ushort4), cudaMemcpyHostToDevice, st);
        if (ce == cudaSuccess) ce = cudaMemcpyAsync(d_row, row.data(), row.size() * 2, cudaMemcpyHostToDevice, st);
        if (ce == cudaSuccess) ce = cudaStreamSynchronize(st);  // the host vectors die with this call
        rd.M = M; rd.N = N;
        rd.nthreads = nthreads_;
        rd.kpp = kpp_;
        rd.L = Lsp; rd.rloc = d_rloc;
        rd.idx = d_idx; rd.owner = d_owner; rd.csr_ptr = d_ptr;
        rd.dest = d_dest; rd.row = d_row; rd.maxval = maxval; rd.Ltot = Ltot;
    };
    ResHost *rh = new ResHost();
    rh->ept = res_ept(M);
    rh->ept_fwd = res_ept_fwd(M, N, d->n_envs);
    build_layout(res_threads(M, rh->ept), rh->rd);
    if (rh->ept_fwd == rh->ept) rh->rd_fwd = rh->rd;
    else build_layout(res_threads(M, rh->ept_fwd), rh->rd_fwd);
    if (ce == cudaSuccess) ce = cudaMemcpyAsync(d_rloc, rloc.data(), rloc.size() * 2, cudaMemcpyHostToDevice, st);
    if (ce == cudaSuccess) ce = cudaMemcpyAsync(d_idx, idx.data(), idx.size() * sizeof(ushort4), cudaMemcpyHostToDevice, st);
    if (ce == cudaSuccess) ce = cudaMemcpyAsync(d_ptr, ptr.data(), ptr.size() * 2, cudaMemcpyHostToDevice, st);
    if (ce == cudaSuccess) ce = cudaStreamSynchronize(st);
    if (ce != cudaSuccess) { delete rh; return cuda_fail(ce, "resident upload"); }
    rh->smem_fwd = res_smem(Lsp, N, rh->rd_fwd.Ltot, rh->rd_fwd.maxval, 1, false);
    rh->smem_adj = res_smem(Lsp, N, rh->rd.Ltot, rh->rd.maxval, 2, true);
    m->res_host = rh;
    int rc = GS_OK;
#define GS_RES_SMEM(K_, E_, T_, B_, BYTES_)                                  \
    do {                                                                     \
        if (rc == GS_OK) rc = set_smem(K_<E_, T_, B_, false>, BYTES_);       \
        if (rc == GS_OK) rc = set_smem(K_<E_, T_, B_, true>, BYTES_);        \
    } while (0)
    if (rh->ept_fwd == 2 && rh->rd_fwd.nthreads <= 160) GS_RES_SMEM(k_resident_fwd, 2, 160, 4, rh->smem_fwd);
    else if (rh->ept_fwd == 1 && rh->rd_fwd.nthreads <= 320) GS_RES_SMEM(k_resident_fwd, 1, 320, 3, rh->smem_fwd);
    else if (rh->ept_fwd == 1) GS_RES_SMEM(k_resident_fwd, 1, 1024, 1, rh->smem_fwd);
    else GS_RES_SMEM(k_resident_fwd, 2, 1024, 1, rh->smem_fwd);
    if (rh->ept == 1 && rh->rd.nthreads <= 320) GS_RES_SMEM(k_resident_adj, 1, 320, 2, rh->smem_adj);
    else if (rh->ept == 1) GS_RES_SMEM(k_resident_adj, 1, 1024, 1, rh->smem_adj);
    else GS_RES_SMEM(k_resident_adj, 2, 1024, 1, rh->smem_adj);
#undef GS_RES_SMEM
    if (rc != GS_OK) return rc;
    m->plan = GS_PLAN_RESIDENT;
    return GS_OK;
}

void resident_release(gs_model *m) {
    delete res_of(m);
    m->res_host = nullptr;
}

static ResAct res_act(const gs_model *m) {
    ResAct ra = {m->d_act[0], m->d_gact[0], m->act_frames, m->act_stride, (size_t)m->E * m->hes[T_TET].cpad};
    return ra;
}

int resident_rollout(gs_model *m, gs_tape *t, cudaStream_t st) {
    ResHost *rh = res_of(m);
    if (!rh) { set_error("resident plan unavailable"); return GS_ESTATE; }
    const dim3 grid(m->E), block(rh->rd_fwd.nthreads);
    const ResAct ra = res_act(m);
    const bool act = m->act_frames > 0;
    cudaEvent_t ta = m->timing ? timing_begin(m, st) : nullptr;
#define GS_RES_FWD(E_, T_, B_)                                                                                                      \
    do {                                                                                                                            \
        if (act) k_resident_fwd<E_, T_, B_, true><<<grid, block, rh->smem_fwd, st>>>(m->dev, rh->rd_fwd, t->base, t->S, t->T, ra);      \
        else k_resident_fwd<E_, T_, B_, false><<<grid, block, rh->smem_fwd, st>>>(m->dev, rh->rd_fwd, t->base, t->S, t->T, ra);         \
    } while (0)
    if (rh->ept_fwd == 2 && rh->rd_fwd.nthreads <= 160) GS_RES_FWD(2, 160, 4);
    else if (rh->ept_fwd == 1 && rh->rd_fwd.nthreads <= 320) GS_RES_FWD(1, 320, 3);
    else if (rh->ept_fwd == 1) GS_RES_FWD(1, 1024, 1);
    else GS_RES_FWD(2, 1024, 1);
#undef GS_RES_FWD
    GS_RES_CHECK("k_resident_fwd");
    if (ta) timing_end(m, GS_K_RESIDENT_FWD, ta, st);
    return GS_OK;
}

int resident_rollout_backward(gs_model *m, gs_tape *t, int n_frames, int frame_stride, const float *d_adj_x_frames, cudaStream_t st) {
    ResHost *rh = res_of(m);
    if (!rh) { set_error("resident plan unavailable"); return GS_ESTATE; }
    const dim3 grid(m->E), block(rh->rd.nthreads);
    const float *fr = n_frames > 0 ? d_adj_x_frames : nullptr;
    const int stride = frame_stride > 0 ? frame_stride : 1;
    const ResAct ra = res_act(m);
    const bool act = m->act_frames > 0;
    cudaEvent_t ta = m->timing ? timing_begin(m, st) : nullptr;
#define GS_RES_ADJ(E_, T_, B_)                                                                                                                                   \
    do {                                                                                                                                                         \
        if (act) k_resident_adj<E_, T_, B_, true><<<grid, block, rh->smem_adj, st>>>(m->dev, rh->rd, t->base, t->S, t->T, m->d_adjx, m->d_adjv, fr, n_frames, stride, ra);  \
        else k_resident_adj<E_, T_, B_, false><<<grid, block, rh->smem_adj, st>>>(m->dev, rh->rd, t->base, t->S, t->T, m->d_adjx, m->d_adjv, fr, n_frames, stride, ra);     \
    } while (0)
    if (rh->ept == 1 && rh->rd.nthreads <= 320) GS_RES_ADJ(1, 320, 2);
    else if (rh->ept == 1) GS_RES_ADJ(1, 1024, 1);
    else GS_RES_ADJ(2, 1024, 1);
#undef GS_RES_ADJ
    GS_RES_CHECK("k_resident_adj");
    if (ta) timing_end(m, GS_K_RESIDENT_ADJ, ta, st);
    return GS_OK;
}

}  // namespace gs
