// gs_internal.h -- host-side model / tape objects and the POD views handed to kernels.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>
#include <string>
#include <vector>

#include "../../include/gradsim.h"

namespace gs {

enum { T_TET = 0, T_TRI = 1, T_HINGE = 2, N_TYPES = 3 };
static const int kArity[N_TYPES] = {4, 3, 4};
static const int kNumGrads[N_TYPES] = {3, 5, 1};  // accumulated parameter gradients per element: tets (mu, lambda, k_damp); triangles the
                                                  // same plus the element's terms of dL/dk_drag, dL/dk_lift (summed per environment on read); hinges k_b

constexpr int kTileElems = 128;      // elements per tile = threads per CTA of the streaming element kernels
constexpr int kConSlots = 64;        // accumulator slots per environment for the per-environment gradient totals
constexpr int kAccVals = 12;         // values per slot: dL/d(k_e, k_d, k_f, mu_c), dL/dg (3), dL/d(k_drag, k_lift), pad
constexpr int kFlushEvery = 32;      // substeps between fp32 -> fp64 parameter-gradient flushes (hazard H4)

// Byte layout of one tile's RECORD: everything static a tile of kTileElems elements needs, packed contiguously so
// that ONE bulk copy (cp.async.bulk, TMA) brings it into shared memory:
//   lidx   ushort4[256]  tile-local particle indices (w unused for triangles)
//   c0     float4[256]   tets: B[0..3]; tris: 2x2 B; hinges: (sin(theta0/2), cos(theta0/2), kb * l0, l0)
//   c1     float4[256]   tets: B[4..7]
//   c2     float2[256]   tets: (B[8], V)
//   area   float[256]    tris: rest area
//   slots     u16[4*128]  gather list: slot = k * 128 + local element of every element-vertex of the tile, sorted by
//                         tile-particle (padded to 4 per element for every type)
//   slot_desc u16[128]    thread t of the CTA sums entries 4t .. 4t+3 and issues one reduction per run of equal
//                         particles (perfectly balanced, no loop); its descriptor packs: bits 0-9 the tile-local
//                         particle of entry 4t, bits 10-12 "entry 4t+k (k = 1..3) starts the next particle" (entries
//                         are sorted, so the next particle is the previous + 1), bits 13-15 the number of valid entries
template <int TYPE>
struct RecLayout {
    static constexpr int kArityT = TYPE == 1 ? 3 : 4;
    static constexpr int oLidx = 0;
    static constexpr int oC0 = kTileElems * 8;
    static constexpr int oC1 = oC0 + kTileElems * 16;
    static constexpr int oC2 = oC1 + (TYPE == 0 ? kTileElems * 16 : 0);
    static constexpr int oArea = oC2 + (TYPE == 0 ? kTileElems * 8 : 0);
    static constexpr int oSlots = oArea + (TYPE == 1 ? kTileElems * 4 : 0);
    static constexpr int oSlotDesc = oSlots + 4 * kTileElems * 2;
    static constexpr int kBytes = oSlotDesc + kTileElems * 2;
};
inline int rec_bytes_of(int type) { return type == 0 ? RecLayout<0>::kBytes : (type == 1 ? RecLayout<1>::kBytes : RecLayout<2>::kBytes); }
constexpr int kParBytes = 3 * kTileElems * 4;  // one tile's (mu | lambda | k_damp) block of one environment

// Device view of one element set (tets, triangles or hinges) in INTERNAL (Morton, tiled) order.
struct ElemDev {
    int count, cpad, n_tiles, pmax;  // cpad = n_tiles * kTileElems; pmax: particle list entries per tile (multiple of 8)
    int lmax;                   // tile-local particle index space (multiple of 8, >= pmax): see tile_parts
    int rec_bytes;              // RecLayout<type>::kBytes
    const char *rec;            // [n_tiles][rec_bytes]
    const int *tile_parts;      // [n_tiles] blocks of { int id[pmax]; uint16_t loc[pmax]; }: the tile's particles, ascending
                                // internal id (-1 padded), and the tile-local index each is staged at.  Local indices are
                                // assigned by colouring: particles read by the same quarter-warp for the same vertex get
                                // different residues mod 8, i.e. different 16-byte bank groups (conflict-free LDS.128)
    float *par;                 // [E][n_tiles][3][kTileElems]  mu, lambda, k_damp (tets, tris)
    float *g32;                 // [kNumGrads][E][cpad] per-substep fp32 accumulators (mu, lambda, damp; hinges: k_b)
    double *g64;                // [kNumGrads][E][cpad] fp64 masters
    const int *perm;            // [count] internal -> caller element index
    const int *det_list;        // deterministic mode (gs_set_deterministic): the tiles of ONE colour class this launch walks
    int det_n;                  //   (no two tiles of a class share a particle); null / 0 in the normal mode
};
// index of parameter q (0 mu, 1 lambda, 2 damp) of internal element e of environment env inside ElemDev::par
__host__ __device__ inline size_t par_index(int n_tiles, int env, int e, int q) {
    return (((size_t)env * n_tiles + (e / kTileElems)) * 3 + q) * kTileElems + (e % kTileElems);
}

struct ModelDev {
    int N, E;
    ElemDev es[N_TYPES];
    float gx, gy, gz, dt;
    float nx, ny, nz, pd, pr;
    const float *ke, *kd, *kf, *muc;  // [E]
    const float *kdrag, *klift;       // [E] lift / drag coefficients of the air (A21)
    float wx, wy, wz;                 // wind
    int aero;                         // some environment has a non-zero air coefficient: the extended element kernels run
    const int *perm_p;                // [N] internal -> caller particle index
    const float *inv_mass;            // [E][N] internal order (0 = pinned)
    float *gmass32;                   // [E][N]
    double *gmass64;                  // [E][N]
    double *gacc;                     // [E][kConSlots][kAccVals] per-environment totals dL/d(k_e, k_d, k_f, mu_c) and dL/dg:
                                      // fp64 partial sums (red.global.add.f64 per warp), spread over slots so that the
                                      // warps of a launch do not all reduce into one L2 sector
    double *gcon64;                   // [E][kAccVals] fp64 masters
    int *tile_ctr;                    // [6] dynamic tile queues of the element kernels: forward tets/tris/hinges, adjoint
                                      // tets/tris/hinges.  Zero between launches: k_particles_fwd re-zeroes the forward
                                      // three after every k_elements_fwd, k_particles_adj the adjoint three before every
                                      // k_elements_adj
    int *bad;                         // first non-finite substep (INT_MAX = none)
    int want_gravity;                 // dL/dg requested (gs_request_grads): the particle adjoint reduces dt lv over all particles
    const float **frame_base;         // [1] base of the caller's frame-cotangent array of the running backward pass: read
                                      // through this slot (written by a one-thread kernel before the pass) so that the
                                      // captured backward graph does not depend on the caller's pointer
};

// Actuation inputs of ONE substep (PAPER.md:579 per-tet, 585-586 per-hinge): the frame of the
// model's activation schedule that holds during this substep, internal element order [E][cpad]; null = passive.
// Passed by value beside ModelDev to the element kernels.
struct ActDev {
    const float *tet, *hinge;  // activation values
    float *g_tet, *g_hinge;    // dL/d(activation) accumulators of the same frame (adjoint kernels)
};

struct HostElemSet {
    int count = 0, cpad = 0, n_tiles = 0, max_tile_parts = 0, pmax = 0, lmax = 0;
    std::vector<int> perm;  // internal -> caller
};

}  // namespace gs

struct gs_model {
    gs::ModelDev dev;
    int N = 0, E = 0, plan = GS_PLAN_STREAMING;
    int counts[gs::N_TYPES] = {0, 0, 0};
    gs::HostElemSet hes[gs::N_TYPES];
    std::vector<int> perm_p;  // internal -> caller
    // scratch device buffers (inside the workspace)
    float4 *d_f = nullptr;                 // [E][N] force accumulators (zero between substeps)
    float4 *d_xs[2] = {nullptr, nullptr};  // single-step state scratch
    float4 *d_vs[2] = {nullptr, nullptr};
    float4 *d_adjx = nullptr, *d_adjv = nullptr, *d_adjf = nullptr;
    // mutable copies of device pointers the API writes
    float *d_inv_mass = nullptr;
    int steps_since_flush = 0;
    int n_sms = 148;
    int smem_fwd = 0, smem_adj = 0;  // dynamic shared memory of the element kernels
    int occ_fwd = 1, occ_adj = 1;    // co-resident CTAs per SM
    bool pdl = true;                 // programmatic dependent launch of the hot-path kernels (small meshes only: configure_stream_kernels)
    long long elem_items = 0;        // work items (tile x environment) of the largest element type
    int step_counter = 0;  // substep index written to dev.bad on a non-finite state
    // activation schedule (gs_actuation_create): n_frames frames of act_stride substeps, [F][E][cpad] per kind (0 tets, 1 hinges)
    int act_frames = 0, act_stride = 1, act_cur = 0;  // act_cur: the frame single-substep calls use
    float *d_act[2] = {nullptr, nullptr}, *d_gact[2] = {nullptr, nullptr};
    gs::ActDev act_for(int substep) const {
        gs::ActDev a = {nullptr, nullptr, nullptr, nullptr};
        if (act_frames <= 0) return a;
        int f = substep / act_stride;
        f = f < act_frames ? f : act_frames - 1;
        const size_t o0 = (size_t)f * E * hes[gs::T_TET].cpad, o1 = (size_t)f * E * hes[gs::T_HINGE].cpad;
        if (counts[gs::T_TET]) { a.tet = d_act[0] + o0; a.g_tet = d_gact[0] + o0; }
        if (counts[gs::T_HINGE]) { a.hinge = d_act[1] + o1; a.g_hinge = d_gact[1] + o1; }
        return a;
    }
    bool aero_host = false;  // build_model: some air coefficient is non-zero
    // deterministic mode: tiles of all element types coloured so that tiles of one colour share no particle; the element
    // kernels are then launched once per colour, and every particle's sum is formed in colour order
    bool det = false;
    int det_colours = 0;
    int *d_det[gs::N_TYPES] = {nullptr, nullptr, nullptr};  // [n_tiles] tile indices sorted by colour
    std::vector<int> det_off[gs::N_TYPES];                  // [det_colours + 1] offsets of the colour classes
    uint64_t epoch = 0;    // bumped when a by-value kernel argument changes (gravity): captured graphs of older epochs are stale
    // resident plan (gs_resident.cu): host descriptor, null when the model runs the streaming plan
    void *res_host = nullptr;
    // per-kernel event timing (gs_kernel_timing)
    bool timing = false;
    std::vector<cudaEvent_t> ev_pool;  // all events ever created for this model
    size_t ev_used = 0;
    struct TimedLaunch { int id; cudaEvent_t a, b; };
    std::vector<TimedLaunch> timed;
    ~gs_model();
};

struct gs_tape {
    gs_model *m = nullptr;
    int T = 0, K = 1, n_ck = 0;
    size_t S = 0;  // float4 elements per array per slot = E * N
    float4 *base = nullptr;
    bool has_rollout = false;
    // CUDA graphs of the streaming plan's launch sequences (the tape slots, and hence every kernel argument, are fixed
    // per tape): captured on a private stream at the first rollout / backward, replayed on the caller's stream
    cudaStream_t cap_stream = nullptr;
    cudaGraphExec_t g_fwd = nullptr, g_bwd = nullptr;
    uint64_t g_fwd_launches = 0, g_bwd_launches = 0;
    int g_bwd_n_frames = -1, g_bwd_stride = 0;  // the backward graph is specific to these frame arguments (not to the pointer)
    bool no_graph = false;                // capture failed once: launch directly from then on
    uint64_t g_epoch = 0;                 // model epoch the graphs were captured at
    ~gs_tape() {
        if (g_fwd) cudaGraphExecDestroy(g_fwd);
        if (g_bwd) cudaGraphExecDestroy(g_bwd);
        if (cap_stream) cudaStreamDestroy(cap_stream);
    }
    // slot index helpers (each slot = x4[S] then v4[S])
    float4 *slot_x(int s) const { return base + (size_t)(2 * s) * S; }
    float4 *slot_v(int s) const { return base + (size_t)(2 * s + 1) * S; }
    int n_slots() const { return K == 1 ? T + 1 : n_ck + 1 + (K - 1 > 2 ? K - 1 : 2); }
    int slot_final() const { return K == 1 ? T : n_ck; }
    int slot_work(int j) const { return n_ck + 1 + j; }  // K > 1 only
    // slot holding state t during the forward pass
    int slot_fwd(int t) const {
        if (K == 1) return t;
        if (t == T) return slot_final();
        if (t % K == 0) return t / K;
        return slot_work(t & 1);
    }
    // slot holding state t while segment c = t0/K is being processed backward (t in [t0, t1])
    int slot_bwd(int t) const {
        if (K == 1) return t;
        if (t == T) return slot_final();
        if (t % K == 0) return t / K;
        return slot_work(t % K - 1);
    }
    bool holds(int t) const { return t >= 0 && t <= T && (K == 1 || t == T || t % K == 0); }
};

namespace gs {
void set_error(const char *fmt, ...);
// event bracket around one launch when m->timing is on (gs_api.cu)
cudaEvent_t timing_begin(gs_model *m, cudaStream_t st);
void timing_end(gs_model *m, int id, cudaEvent_t a, cudaStream_t st);
int cuda_fail(cudaError_t e, const char *what);
extern std::atomic<uint64_t> g_launches;  // process-wide launch counter (models on different host threads share it)
extern thread_local bool t_capturing;     // this host thread is capturing a CUDA graph: launches are counted into t_captured
extern thread_local uint64_t t_captured;
inline void count_launch(uint64_t n = 1) {
    if (t_capturing) t_captured += n;
    else g_launches.fetch_add(n, std::memory_order_relaxed);
}

// gs_plan.cpp: host preprocessing.  Fills a byte image of the workspace (static part) and the model's host fields.
struct WorkspaceLayout;
size_t workspace_bytes_upper(int N, int E, const int counts[N_TYPES]);
int build_model(const gs_model_desc *desc, void *d_workspace, size_t bytes, cudaStream_t stream, gs_model *m);

// gs_stream.cu: streaming plan launches
int stream_step_forward(gs_model *m, const float4 *x, const float4 *v, float4 *xo, float4 *vo, int substep, cudaStream_t st);
int stream_step_adjoint(gs_model *m, const float4 *x, const float4 *v, const float4 *v_next, long long frame_off, int substep, cudaStream_t st);
int launch_set_frame_base(gs_model *m, const float *d_frames, cudaStream_t st);
int launch_pack(gs_model *m, const float *x, const float *v, float4 *x4, float4 *v4, bool x_is_state, cudaStream_t st);
int launch_unpack(gs_model *m, const float4 *x4, const float4 *v4, float *x, float *v, cudaStream_t st);
int launch_flush_grads(gs_model *m, cudaStream_t st);
int launch_zero_grads(gs_model *m, cudaStream_t st);
int launch_get_grads(gs_model *m, int group, float *d_out, cudaStream_t st);
int launch_set_params(gs_model *m, int group, const float *d_values, cudaStream_t st);
int launch_actuation_io(gs_model *m, int kind, const float *d_in, float *d_out, cudaStream_t st);  // caller order <-> internal schedule
int configure_stream_kernels(gs_model *m);

// gs_resident.cu: resident plan
size_t resident_blob_bytes(const gs_model_desc *desc);
int resident_prepare(gs_model *m, const gs_model_desc *desc, void *d_workspace, size_t bytes, cudaStream_t st);
void resident_release(gs_model *m);
int resident_rollout(gs_model *m, gs_tape *t, cudaStream_t st);
int resident_rollout_backward(gs_model *m, gs_tape *t, int n_frames, int frame_stride, const float *d_adj_x_frames, cudaStream_t st);
}  // namespace gs
