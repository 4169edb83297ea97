// gs_api.cu -- extern "C" entry points of include/gradsim.h: argument checks, tape bookkeeping, rollout /
// backward drivers (streaming or resident plan), loss helpers, host-buffer end-to-end call.
#include <climits>
#include <cstring>
#include <new>

#include "gs_internal.h"

using namespace gs;

namespace gs {
const char *last_error();
}

#define GS_REQUIRE(cond, code, ...)      \
    do {                                 \
        if (!(cond)) {                   \
            set_error(__VA_ARGS__);      \
            return code;                 \
        }                                \
    } while (0)
#define GS_TRY(expr)                     \
    do {                                 \
        int rc_ = (expr);                \
        if (rc_ != GS_OK) return rc_;    \
    } while (0)
#define GS_CUDA(expr, what)                                   \
    do {                                                      \
        cudaError_t e_ = (expr);                              \
        if (e_ != cudaSuccess) return cuda_fail(e_, what);    \
    } while (0)

static int check_desc(const gs_model_desc *d) {
    GS_REQUIRE(d, GS_EINVAL, "desc is null");
    GS_REQUIRE(d->n_particles > 0 && d->n_envs > 0, GS_EINVAL, "n_particles and n_envs must be > 0");
    GS_REQUIRE(d->n_tets >= 0 && d->n_tris >= 0 && d->n_hinges >= 0, GS_EINVAL, "negative element count");
    GS_REQUIRE(d->x_rest && d->mass, GS_EINVAL, "x_rest and mass are required");
    GS_REQUIRE(d->n_tets == 0 || (d->tets && d->tet_mu && d->tet_lambda && d->tet_damp), GS_EINVAL, "tet arrays missing");
    GS_REQUIRE(d->n_tris == 0 || (d->tris && d->tri_mu && d->tri_lambda && d->tri_damp), GS_EINVAL, "triangle arrays missing");
    GS_REQUIRE(d->n_hinges == 0 || (d->hinges && d->hinge_kb), GS_EINVAL, "hinge arrays missing");
    GS_REQUIRE(d->ke && d->kd && d->kf && d->mu_c, GS_EINVAL, "contact parameters missing");
    GS_REQUIRE(d->dt > 0.0f, GS_EINVAL, "dt must be > 0");
    GS_REQUIRE(d->plan >= GS_PLAN_AUTO && d->plan <= GS_PLAN_RESIDENT, GS_EINVAL, "unknown plan %d", d->plan);
    GS_REQUIRE((size_t)d->n_particles * (size_t)d->n_envs < ((size_t)1 << 31), GS_EINVAL, "E*N must be < 2^31");
    {  // work items (tile x environment) and padded element counts are ints in the kernels
        const long long mx = d->n_tets > d->n_tris ? (d->n_tets > d->n_hinges ? d->n_tets : d->n_hinges) : (d->n_tris > d->n_hinges ? d->n_tris : d->n_hinges);
        GS_REQUIRE((mx + kTileElems) * (long long)d->n_envs < (1LL << 31), GS_EINVAL, "E * padded element count must be < 2^31");
    }
    return GS_OK;
}

extern "C" size_t gs_model_workspace_bytes(const gs_model_desc *d) {
    if (check_desc(d) != GS_OK) return 0;
    const int counts[N_TYPES] = {d->n_tets, d->n_tris, d->n_hinges};
    return workspace_bytes_upper(d->n_particles, d->n_envs, counts) + resident_blob_bytes(d);
}

extern "C" int gs_model_create(const gs_model_desc *d, void *d_workspace, size_t bytes, gs_stream stream, gs_model **out) {
    GS_REQUIRE(out, GS_EINVAL, "out is null");
    *out = nullptr;
    GS_TRY(check_desc(d));
    GS_REQUIRE(d_workspace, GS_EINVAL, "workspace is null");
    gs_model *m = new (std::nothrow) gs_model();
    GS_REQUIRE(m, GS_ENOMEM, "out of host memory");
    int rc = GS_OK;
    try {
        rc = build_model(d, d_workspace, bytes, (cudaStream_t)stream, m);
        if (rc == GS_OK) rc = configure_stream_kernels(m);
        if (rc == GS_OK) rc = resident_prepare(m, d, d_workspace, bytes, (cudaStream_t)stream);
    } catch (const std::bad_alloc &) {
        set_error("out of host memory while planning the model");
        rc = GS_ENOMEM;
    }
    if (rc != GS_OK) { delete m; return rc; }
    *out = m;
    return GS_OK;
}

extern "C" void gs_model_destroy(gs_model *m) { delete m; }
extern "C" int gs_model_plan(const gs_model *m) { return m ? m->plan : GS_EINVAL; }
extern "C" int gs_model_info(const gs_model *m, int32_t *n_particles, int32_t *n_elements, int32_t *n_envs) {
    GS_REQUIRE(m, GS_EINVAL, "model is null");
    if (n_particles) *n_particles = m->N;
    if (n_elements) *n_elements = m->counts[0] + m->counts[1] + m->counts[2];
    if (n_envs) *n_envs = m->E;
    return GS_OK;
}

extern "C" int gs_set_params(gs_model *m, int group, const float *d_values, gs_stream stream) {
    GS_REQUIRE(m && d_values, GS_EINVAL, "null argument");
    GS_REQUIRE(group >= 0 && group < GS_NUM_GROUPS, GS_EINVAL, "unknown parameter group %d", group);
    return launch_set_params(m, group, d_values, (cudaStream_t)stream);
}

// ------------------------------------------------------------------------------------------ actuation inputs
static size_t act_floats(const gs_model *m, int kind, int n_frames) {
    const int t = kind == 0 ? T_TET : T_HINGE;
    return m->counts[t] ? (size_t)n_frames * m->E * m->hes[t].cpad : 0;
}
static size_t al256f(size_t n) { return (n + 63) & ~(size_t)63; }  // floats, 256-byte granules
extern "C" size_t gs_actuation_bytes(const gs_model *m, int n_frames) {
    if (!m || n_frames < 1) return 0;
    return 2 * (al256f(act_floats(m, 0, n_frames)) + al256f(act_floats(m, 1, n_frames))) * sizeof(float) + 256;
}
extern "C" int gs_actuation_create(gs_model *m, int n_frames, int frame_stride, void *d_mem, size_t bytes, gs_stream stream) {
    GS_REQUIRE(m, GS_EINVAL, "model is null");
    m->epoch++;  // the frame pointers are kernel arguments: captured graphs are stale
    m->act_cur = 0;
    if (n_frames == 0) { m->act_frames = 0; m->d_act[0] = m->d_act[1] = m->d_gact[0] = m->d_gact[1] = nullptr; return GS_OK; }
    GS_REQUIRE(n_frames >= 1 && frame_stride >= 1, GS_EINVAL, "n_frames and frame_stride must be >= 1");
    GS_REQUIRE(d_mem && ((uintptr_t)d_mem & 255) == 0 && bytes >= gs_actuation_bytes(m, n_frames), GS_EINVAL, "actuation memory missing, misaligned or too small (%zu < %zu)",
               bytes, gs_actuation_bytes(m, n_frames));
    float *p = (float *)d_mem;
    for (int k = 0; k < 2; k++) { m->d_act[k] = p; p += al256f(act_floats(m, k, n_frames)); m->d_gact[k] = p; p += al256f(act_floats(m, k, n_frames)); }
    GS_CUDA(cudaMemsetAsync(d_mem, 0, gs_actuation_bytes(m, n_frames) - 256, (cudaStream_t)stream), "zero actuation memory");
    m->act_frames = n_frames; m->act_stride = frame_stride;
    return GS_OK;
}
extern "C" int gs_set_actuation(gs_model *m, int kind, const float *d_values, gs_stream stream) {
    GS_REQUIRE(m && d_values, GS_EINVAL, "null argument");
    GS_REQUIRE(kind == GS_ACT_TET || kind == GS_ACT_HINGE, GS_EINVAL, "unknown actuation kind %d", kind);
    GS_REQUIRE(m->act_frames > 0, GS_ESTATE, "no activation schedule attached (gs_actuation_create)");
    return launch_actuation_io(m, kind, d_values, nullptr, (cudaStream_t)stream);
}
extern "C" int gs_actuation_grads(gs_model *m, int kind, float *d_out, gs_stream stream) {
    GS_REQUIRE(m && d_out, GS_EINVAL, "null argument");
    GS_REQUIRE(kind == GS_ACT_TET || kind == GS_ACT_HINGE, GS_EINVAL, "unknown actuation kind %d", kind);
    GS_REQUIRE(m->act_frames > 0, GS_ESTATE, "no activation schedule attached (gs_actuation_create)");
    return launch_actuation_io(m, kind, nullptr, d_out, (cudaStream_t)stream);
}
extern "C" int gs_set_actuation_frame(gs_model *m, int frame) {
    GS_REQUIRE(m, GS_EINVAL, "model is null");
    GS_REQUIRE(m->act_frames > 0 && frame >= 0 && frame < m->act_frames, GS_EINVAL, "frame %d outside the schedule of %d frames", frame, m->act_frames);
    m->act_cur = frame;
    return GS_OK;
}

extern "C" int gs_request_grads(gs_model *m, int group, int enable) {
    GS_REQUIRE(m, GS_EINVAL, "model is null");
    GS_REQUIRE(group == GS_GRAVITY, GS_EINVAL, "group %d needs no request: only GS_GRAVITY is off by default", group);
    if (m->dev.want_gravity != (enable != 0)) { m->dev.want_gravity = enable != 0; m->epoch++; }  // a by-value kernel argument
    return GS_OK;
}

extern "C" int gs_set_deterministic(gs_model *m, int enable) {
    GS_REQUIRE(m, GS_EINVAL, "model is null");
    GS_REQUIRE(!enable || m->det_colours > 0, GS_ESTATE, "the mesh's tiles need more than 64 colours: no deterministic mode for this model");
    if (m->det != (enable != 0)) { m->det = enable != 0; m->epoch++; }
    return GS_OK;
}

static int reset_bad(gs_model *m, cudaStream_t st) {
    GS_CUDA(cudaMemsetAsync(m->dev.bad, 0x7f, sizeof(int), st), "reset non-finite flag");
    return GS_OK;
}

extern "C" int gs_step_forward(gs_model *m, const float *d_x, const float *d_v, float *d_x_out, float *d_v_out, gs_stream stream) {
    GS_REQUIRE(m && d_x && d_v && d_x_out && d_v_out, GS_EINVAL, "null argument");
    cudaStream_t st = (cudaStream_t)stream;
    GS_TRY(reset_bad(m, st));
    GS_TRY(launch_pack(m, d_x, d_v, m->d_xs[0], m->d_vs[0], true, st));
    GS_TRY(stream_step_forward(m, m->d_xs[0], m->d_vs[0], m->d_xs[1], m->d_vs[1], -1, st));
    return launch_unpack(m, m->d_xs[1], m->d_vs[1], d_x_out, d_v_out, st);
}

extern "C" int gs_step_backward(gs_model *m, const float *d_x, const float *d_v, const float *d_adj_x_out, const float *d_adj_v_out,
                                float *d_adj_x_in, float *d_adj_v_in, gs_stream stream) {
    GS_REQUIRE(m && d_x && d_v && d_adj_x_out && d_adj_v_out && d_adj_x_in && d_adj_v_in, GS_EINVAL, "null argument");
    cudaStream_t st = (cudaStream_t)stream;
    GS_TRY(reset_bad(m, st));
    GS_TRY(launch_pack(m, d_x, d_v, m->d_xs[0], m->d_vs[0], true, st));
    // the end-of-step velocity enters the mass gradient: recompute the forward step
    GS_TRY(stream_step_forward(m, m->d_xs[0], m->d_vs[0], m->d_xs[1], m->d_vs[1], -1, st));
    GS_TRY(launch_pack(m, d_adj_x_out, d_adj_v_out, m->d_adjx, m->d_adjv, false, st));
    GS_TRY(stream_step_adjoint(m, m->d_xs[0], m->d_vs[0], m->d_vs[1], -1, -1, st));
    return launch_unpack(m, m->d_adjx, m->d_adjv, d_adj_x_in, d_adj_v_in, st);
}

// ------------------------------------------------------------------------------------------ tape
static int tape_slots(int T, int K) {
    if (K == 1) return T + 1;
    const int n_ck = (T + K - 1) / K;
    return n_ck + 1 + (K - 1 > 2 ? K - 1 : 2);
}

extern "C" size_t gs_tape_bytes(const gs_model *m, int n_substeps, int checkpoint_every) {
    if (!m || n_substeps < 1 || checkpoint_every < 1) return 0;
    const int K = checkpoint_every > n_substeps ? n_substeps : checkpoint_every;
    return (size_t)tape_slots(n_substeps, K) * 2 * (size_t)m->E * m->N * sizeof(float4) + 256;
}

extern "C" int gs_tape_create(gs_model *m, int n_substeps, int checkpoint_every, void *d_mem, size_t bytes, gs_tape **out) {
    GS_REQUIRE(out, GS_EINVAL, "out is null");
    *out = nullptr;
    GS_REQUIRE(m && d_mem, GS_EINVAL, "null argument");
    GS_REQUIRE(n_substeps >= 1 && checkpoint_every >= 1, GS_EINVAL, "n_substeps and checkpoint_every must be >= 1");
    GS_REQUIRE(((uintptr_t)d_mem & 255) == 0, GS_EINVAL, "tape memory must be 256-byte aligned");
    GS_REQUIRE(bytes >= gs_tape_bytes(m, n_substeps, checkpoint_every), GS_EINVAL, "tape memory too small: %zu < %zu", bytes,
               gs_tape_bytes(m, n_substeps, checkpoint_every));
    gs_tape *t = new (std::nothrow) gs_tape();
    GS_REQUIRE(t, GS_ENOMEM, "out of host memory");
    t->m = m; t->T = n_substeps;
    t->K = checkpoint_every > n_substeps ? n_substeps : checkpoint_every;
    t->n_ck = (t->T + t->K - 1) / t->K;
    t->S = (size_t)m->E * m->N;
    t->base = (float4 *)d_mem;
    *out = t;
    return GS_OK;
}
extern "C" void gs_tape_destroy(gs_tape *t) { delete t; }

// Runs `body(stream)` (a fixed sequence of kernel launches) through a CUDA graph: captured once on the tape's private
// stream, then replayed on the caller's stream -- for small meshes the rollout is bound by per-launch latency
// (SURVEY.md 8(a) a7 / north_star (6)).  Falls back to direct launches while per-kernel timing is on or if capture fails.
template <class F>
static int graph_run(gs_model *m, gs_tape *t, cudaGraphExec_t *exec, uint64_t *n_launch, cudaStream_t st, F body) {
    if (m->timing || t->no_graph) return body(st);
    if (*exec && t->g_epoch != m->epoch) {  // a by-value kernel argument (gravity) changed since the capture
        if (t->g_fwd) { cudaGraphExecDestroy(t->g_fwd); t->g_fwd = nullptr; }
        if (t->g_bwd) { cudaGraphExecDestroy(t->g_bwd); t->g_bwd = nullptr; }
    }
    if (!*exec) {
        if (!t->g_fwd && !t->g_bwd) t->g_epoch = m->epoch;
        cudaGraph_t g = nullptr;
        bool ok = t->cap_stream || cudaStreamCreateWithFlags(&t->cap_stream, cudaStreamNonBlocking) == cudaSuccess;
        ok = ok && cudaStreamBeginCapture(t->cap_stream, cudaStreamCaptureModeThreadLocal) == cudaSuccess;
        int rc = GS_OK;
        if (ok) {
            t_capturing = true; t_captured = 0;  // launches enqueued while capturing are counted per replay, not now
            rc = body(t->cap_stream);
            t_capturing = false;
            ok = cudaStreamEndCapture(t->cap_stream, &g) == cudaSuccess && g != nullptr && rc == GS_OK;
        }
        if (ok) {
            *n_launch = t_captured;
            ok = cudaGraphInstantiate(exec, g, 0) == cudaSuccess;
        }
        if (g) cudaGraphDestroy(g);
        if (!ok) {
            cudaGetLastError();
            *exec = nullptr;
            t->no_graph = true;
            return rc != GS_OK ? rc : body(st);
        }
    }
    GS_CUDA(cudaGraphLaunch(*exec, st), "cudaGraphLaunch");
    count_launch(*n_launch);
    return GS_OK;
}

extern "C" int gs_rollout(gs_model *m, gs_tape *t, const float *d_x0, const float *d_v0, float *d_x_T, float *d_v_T, gs_stream stream) {
    GS_REQUIRE(m && t && d_x0 && d_v0, GS_EINVAL, "null argument");
    GS_REQUIRE(t->m == m, GS_EINVAL, "tape belongs to another model");
    cudaStream_t st = (cudaStream_t)stream;
    GS_TRY(reset_bad(m, st));
    GS_TRY(launch_pack(m, d_x0, d_v0, t->slot_x(t->slot_fwd(0)), t->slot_v(t->slot_fwd(0)), true, st));
    if (m->plan == GS_PLAN_RESIDENT && t->K == 1) {  // a checkpointed tape of a resident model runs the streaming loop
        GS_TRY(resident_rollout(m, t, st));
    } else {
        GS_TRY(graph_run(m, t, &t->g_fwd, &t->g_fwd_launches, st, [&](cudaStream_t q) {
            for (int s = 0; s < t->T; s++) {
                const int a = t->slot_fwd(s), b = t->slot_fwd(s + 1);
                GS_TRY(stream_step_forward(m, t->slot_x(a), t->slot_v(a), t->slot_x(b), t->slot_v(b), s, q));
            }
            return (int)GS_OK;
        }));
    }
    t->has_rollout = true;
    return launch_unpack(m, t->slot_x(t->slot_final()), t->slot_v(t->slot_final()), d_x_T, d_v_T, st);
}

extern "C" int gs_tape_read(gs_model *m, gs_tape *t, int substep, float *d_x, float *d_v, gs_stream stream) {
    GS_REQUIRE(m && t && t->m == m, GS_EINVAL, "bad model / tape");
    GS_REQUIRE(t->has_rollout, GS_ESTATE, "the tape holds no rollout yet");
    GS_REQUIRE(t->holds(substep), GS_ESTATE, "the tape does not hold substep %d (T = %d, checkpoint_every = %d)", substep, t->T, t->K);
    const int s = t->slot_bwd(substep);
    return launch_unpack(m, t->slot_x(s), t->slot_v(s), d_x, d_v, (cudaStream_t)stream);
}

extern "C" int gs_rollout_backward(gs_model *m, gs_tape *t, int n_frames, int frame_stride, const float *d_adj_x_frames,
                                   const float *d_adj_x_T, const float *d_adj_v_T, float *d_adj_x0, float *d_adj_v0, gs_stream stream) {
    GS_REQUIRE(m && t && t->m == m, GS_EINVAL, "bad model / tape");
    GS_REQUIRE(t->has_rollout, GS_ESTATE, "gs_rollout_backward needs a gs_rollout on this tape first");
    GS_REQUIRE(n_frames >= 0 && (n_frames == 0 || (d_adj_x_frames && frame_stride >= 1)), GS_EINVAL, "bad frame arguments");
    GS_REQUIRE(n_frames == 0 || (long long)n_frames * frame_stride <= t->T, GS_EINVAL, "frames reach beyond the rollout: %d * %d > %d", n_frames,
               frame_stride, t->T);
    cudaStream_t st = (cudaStream_t)stream;
    GS_TRY(launch_pack(m, d_adj_x_T, d_adj_v_T, m->d_adjx, m->d_adjv, false, st));
    const size_t frame_elems = (size_t)m->E * m->N * 3;
    if (m->plan == GS_PLAN_RESIDENT && t->K == 1) {
        GS_TRY(resident_rollout_backward(m, t, n_frames, frame_stride, d_adj_x_frames, st));
    } else {
        if (t->g_bwd && (t->g_bwd_n_frames != n_frames || t->g_bwd_stride != frame_stride)) {
            cudaGraphExecDestroy(t->g_bwd);  // other frame layout: capture again
            t->g_bwd = nullptr;
        }
        t->g_bwd_n_frames = n_frames; t->g_bwd_stride = frame_stride;
        // the frame array's base pointer reaches the kernels through a workspace slot, so another buffer of the same
        // layout (torch hands out a new address every iteration) replays the same graph
        if (n_frames > 0) GS_TRY(launch_set_frame_base(m, d_adj_x_frames, st));
        GS_TRY(graph_run(m, t, &t->g_bwd, &t->g_bwd_launches, st, [&](cudaStream_t q) {
            GS_TRY(launch_flush_grads(m, q));  // fixed flush positions whatever ran before (resets the 32-substep counter)
            for (int c = t->n_ck - 1; c >= 0; c--) {
                const int t0 = c * t->K, t1 = t0 + t->K < t->T ? t0 + t->K : t->T;
                for (int s = t0; s + 1 < t1; s++) {  // regenerate the segment's states from its checkpoint
                    const int a = t->slot_bwd(s), b = t->slot_bwd(s + 1);
                    GS_TRY(stream_step_forward(m, t->slot_x(a), t->slot_v(a), t->slot_x(b), t->slot_v(b), s, q));
                }
                for (int s = t1 - 1; s >= t0; s--) {
                    long long cot = -1;
                    if (n_frames > 0 && (s + 1) % frame_stride == 0 && (s + 1) / frame_stride <= n_frames)
                        cot = (long long)((s + 1) / frame_stride - 1) * (long long)frame_elems;
                    const int a = t->slot_bwd(s), b = t->slot_bwd(s + 1);
                    GS_TRY(stream_step_adjoint(m, t->slot_x(a), t->slot_v(a), t->slot_v(b), cot, s, q));
                }
            }
            return (int)GS_OK;
        }));
    }
    GS_TRY(launch_flush_grads(m, st));
    return launch_unpack(m, m->d_adjx, m->d_adjv, d_adj_x0, d_adj_v0, st);
}

extern "C" int gs_zero_grads(gs_model *m, gs_stream stream) {
    GS_REQUIRE(m, GS_EINVAL, "model is null");
    return launch_zero_grads(m, (cudaStream_t)stream);
}
extern "C" int gs_param_grads(gs_model *m, int group, float *d_out, gs_stream stream) {
    GS_REQUIRE(m && d_out, GS_EINVAL, "null argument");
    GS_REQUIRE(group >= 0 && group < GS_NUM_GROUPS, GS_EINVAL, "unknown parameter group %d", group);
    GS_REQUIRE(group != GS_WIND, GS_EINVAL, "the wind has no gradient");
    GS_REQUIRE(group != GS_GRAVITY || m->dev.want_gravity, GS_ESTATE, "dL/dg was not requested before the backward pass (gs_request_grads)");
    return launch_get_grads(m, group, d_out, (cudaStream_t)stream);
}

extern "C" int gs_check_finite(gs_model *m, gs_stream stream, int *first_bad_substep) {
    GS_REQUIRE(m, GS_EINVAL, "model is null");
    int bad = 0;
    GS_CUDA(cudaMemcpyAsync(&bad, m->dev.bad, sizeof(int), cudaMemcpyDeviceToHost, (cudaStream_t)stream), "read non-finite flag");
    GS_CUDA(cudaStreamSynchronize((cudaStream_t)stream), "synchronize");
    const bool is_bad = bad >= 0 && bad < 0x7f000000;
    if (first_bad_substep) *first_bad_substep = is_bad ? bad : -1;
    if (is_bad) { set_error("non-finite state first produced by substep %d", bad); return GS_ENONFINITE; }
    return GS_OK;
}

// ------------------------------------------------------------------------------------------ losses
// one CTA per environment
__global__ void __launch_bounds__(1024) k_loss_centroid(int N, const float *__restrict__ x, const float *__restrict__ target, float scale, int accumulate,
                                                       float *__restrict__ loss, float *__restrict__ adj) {
    __shared__ float red[3][32];
    __shared__ float cen[3];
    const int env = blockIdx.x, tid = threadIdx.x;
    const float *xe = x + (size_t)env * N * 3;
    float sx = 0.f, sy = 0.f, sz = 0.f;
    for (int i = tid; i < N; i += blockDim.x) { sx += xe[3 * i]; sy += xe[3 * i + 1]; sz += xe[3 * i + 2]; }
    for (int o = 16; o > 0; o >>= 1) { sx += __shfl_xor_sync(0xffffffffu, sx, o); sy += __shfl_xor_sync(0xffffffffu, sy, o); sz += __shfl_xor_sync(0xffffffffu, sz, o); }
    if ((tid & 31) == 0) { red[0][tid >> 5] = sx; red[1][tid >> 5] = sy; red[2][tid >> 5] = sz; }
    __syncthreads();
    if (tid < 3) {
        float s = 0.f;
        for (int w = 0; w < (int)(blockDim.x >> 5); w++) s += red[tid][w];
        cen[tid] = s / (float)N - target[env * 3 + tid];
    }
    __syncthreads();
    if (tid == 0) {
        const float L = scale * (cen[0] * cen[0] + cen[1] * cen[1] + cen[2] * cen[2]);
        loss[env] = accumulate ? loss[env] + L : L;
    }
    if (adj) {
        const float k = 2.0f * scale / (float)N;
        float *ae = adj + (size_t)env * N * 3;
        for (int i = tid; i < 3 * N; i += blockDim.x) ae[i] = k * cen[i % 3];
    }
}
__global__ void __launch_bounds__(1024) k_loss_pos(int N, const float *__restrict__ x, const float *__restrict__ ref, float scale, int accumulate,
                                                  float *__restrict__ loss, float *__restrict__ adj) {
    __shared__ float red[32];
    const int env = blockIdx.x, tid = threadIdx.x;
    const size_t o = (size_t)env * N * 3;
    float s = 0.f;
    for (int i = tid; i < 3 * N; i += blockDim.x) {
        const float dlt = x[o + i] - ref[o + i];
        s = fmaf(dlt, dlt, s);
        if (adj) adj[o + i] = 2.0f * scale * dlt;
    }
    for (int k = 16; k > 0; k >>= 1) s += __shfl_xor_sync(0xffffffffu, s, k);
    if ((tid & 31) == 0) red[tid >> 5] = s;
    __syncthreads();
    if (tid == 0) {
        float tot = 0.f;
        for (int w = 0; w < (int)(blockDim.x >> 5); w++) tot += red[w];
        tot *= scale;
        loss[env] = accumulate ? loss[env] + tot : tot;
    }
}

// ---- large meshes: the same losses over many CTAs per environment (one CTA per environment leaves 147 SMs idle on a
// 476 k-particle scene).  No scratch memory exists (the library allocates nothing), so the centroid's partial sums
// travel through the TAIL of the adj_x output itself: pass A writes kLossParts partial sums there, pass B (all CTAs) reads
// them, finishes loss and cotangent everywhere except that tail, pass C (one CTA per environment) reads the partials
// into registers, synchronises, and only then overwrites the tail with the cotangent.
constexpr int kLossParts = 128;     // CTAs per environment
constexpr int kLossMinN = 32768;    // below this one CTA per environment is faster than three launches

__device__ __forceinline__ void block_sum3(float &sx, float &sy, float &sz, float (*red)[32]) {
    const int tid = threadIdx.x;
    for (int o = 16; o > 0; o >>= 1) { sx += __shfl_xor_sync(0xffffffffu, sx, o); sy += __shfl_xor_sync(0xffffffffu, sy, o); sz += __shfl_xor_sync(0xffffffffu, sz, o); }
    if ((tid & 31) == 0) { red[0][tid >> 5] = sx; red[1][tid >> 5] = sy; red[2][tid >> 5] = sz; }
    __syncthreads();
    if (tid < 3) {
        float s = 0.f;
        for (int w = 0; w < (int)(blockDim.x >> 5); w++) s += red[tid][w];
        red[tid][0] = s;
    }
    __syncthreads();
    sx = red[0][0]; sy = red[1][0]; sz = red[2][0];
}
// particles [lo, hi) of part b
__device__ __forceinline__ void part_range(int N, int b, int &lo, int &hi) {
    const int per = (N + kLossParts - 1) / kLossParts;
    lo = b * per < N ? b * per : N;
    hi = lo + per < N ? lo + per : N;
}
__global__ void __launch_bounds__(256) k_centroid_partial(int N, const float *__restrict__ x, float *__restrict__ adj) {
    __shared__ float red[3][32];
    const int env = blockIdx.y, b = blockIdx.x;
    int lo, hi;
    part_range(N, b, lo, hi);
    const float *xe = x + (size_t)env * N * 3;
    float sx = 0.f, sy = 0.f, sz = 0.f;
    for (int i = lo + threadIdx.x; i < hi; i += blockDim.x) { sx += xe[3 * i]; sy += xe[3 * i + 1]; sz += xe[3 * i + 2]; }
    block_sum3(sx, sy, sz, red);
    if (threadIdx.x < 3) adj[(size_t)env * N * 3 + (size_t)3 * N - 3 * kLossParts + 3 * b + threadIdx.x] = threadIdx.x == 0 ? sx : (threadIdx.x == 1 ? sy : sz);
}
// tail_only = 0: every CTA finishes the centroid from the partials and writes its particles' cotangent except the tail;
// tail_only = 1 (grid.x = 1): reads the partials, then overwrites the tail
__global__ void __launch_bounds__(256) k_centroid_finish(int N, const float *__restrict__ target, float scale, int accumulate, float *__restrict__ loss,
                                                         float *__restrict__ adj, int tail_only) {
    __shared__ float cen[3];
    const int env = blockIdx.y, b = blockIdx.x, tid = threadIdx.x;
    float *ae = adj + (size_t)env * N * 3;
    const size_t tail = (size_t)3 * N - 3 * kLossParts;
    if (tid < 3) {
        float s = 0.f;
        for (int q = 0; q < kLossParts; q++) s += ae[tail + 3 * q + tid];
        cen[tid] = s / (float)N - target[env * 3 + tid];
    }
    __syncthreads();
    const float k = 2.0f * scale / (float)N;
    if (tail_only) {
        for (size_t i = tail + tid; i < (size_t)3 * N; i += blockDim.x) ae[i] = k * cen[i % 3];
        return;
    }
    if (b == 0 && tid == 0) {
        const float L = scale * (cen[0] * cen[0] + cen[1] * cen[1] + cen[2] * cen[2]);
        loss[env] = accumulate ? loss[env] + L : L;
    }
    int lo, hi;
    part_range(N, b, lo, hi);
    for (size_t i = (size_t)3 * lo + tid; i < (size_t)3 * hi && i < tail; i += blockDim.x) ae[i] = k * cen[i % 3];
}
__global__ void __launch_bounds__(256) k_loss_pos_parts(int N, const float *__restrict__ x, const float *__restrict__ ref, float scale,
                                                        float *__restrict__ loss, float *__restrict__ adj) {
    __shared__ float red[3][32];
    const int env = blockIdx.y, b = blockIdx.x;
    int lo, hi;
    part_range(N, b, lo, hi);
    const size_t o = (size_t)env * N * 3;
    float s = 0.f, u = 0.f, w = 0.f;
    for (size_t i = (size_t)3 * lo + threadIdx.x; i < (size_t)3 * hi; i += blockDim.x) {
        const float dlt = x[o + i] - ref[o + i];
        s = fmaf(dlt, dlt, s);
        if (adj) adj[o + i] = 2.0f * scale * dlt;
    }
    block_sum3(s, u, w, red);
    if (threadIdx.x == 0) atomicAdd(loss + env, scale * s);
}

extern "C" int gs_loss_centroid(int n_envs, int n_particles, const float *d_x, const float *d_target, float scale, int accumulate, float *d_loss,
                                float *d_adj_x, gs_stream stream) {
    GS_REQUIRE(n_envs > 0 && n_particles > 0 && d_x && d_target && d_loss, GS_EINVAL, "bad argument");
    if (n_particles >= kLossMinN && d_adj_x && n_envs <= 65535) {
        cudaStream_t st = (cudaStream_t)stream;
        k_centroid_partial<<<dim3(kLossParts, n_envs), 256, 0, st>>>(n_particles, d_x, d_adj_x);
        k_centroid_finish<<<dim3(kLossParts, n_envs), 256, 0, st>>>(n_particles, d_target, scale, accumulate, d_loss, d_adj_x, 0);
        k_centroid_finish<<<dim3(1, n_envs), 256, 0, st>>>(n_particles, d_target, scale, accumulate, d_loss, d_adj_x, 1);
        GS_CUDA(cudaGetLastError(), "k_centroid_partial / k_centroid_finish");
        count_launch(3);
        return GS_OK;
    }
    k_loss_centroid<<<n_envs, n_particles >= 4096 ? 1024 : 256, 0, (cudaStream_t)stream>>>(n_particles, d_x, d_target, scale, accumulate, d_loss, d_adj_x);
    GS_CUDA(cudaGetLastError(), "k_loss_centroid");
    count_launch();
    return GS_OK;
}
extern "C" int gs_loss_pos(int n_envs, int n_particles, const float *d_x, const float *d_ref, float scale, int accumulate, float *d_loss, float *d_adj_x,
                           gs_stream stream) {
    GS_REQUIRE(n_envs > 0 && n_particles > 0 && d_x && d_ref && d_loss, GS_EINVAL, "bad argument");
    if (n_particles >= kLossMinN && n_envs <= 65535) {
        cudaStream_t st = (cudaStream_t)stream;
        if (!accumulate) GS_CUDA(cudaMemsetAsync(d_loss, 0, sizeof(float) * (size_t)n_envs, st), "zero loss");
        k_loss_pos_parts<<<dim3(kLossParts, n_envs), 256, 0, st>>>(n_particles, d_x, d_ref, scale, d_loss, d_adj_x);
        GS_CUDA(cudaGetLastError(), "k_loss_pos_parts");
        count_launch();
        return GS_OK;
    }
    k_loss_pos<<<n_envs, n_particles >= 4096 ? 1024 : 256, 0, (cudaStream_t)stream>>>(n_particles, d_x, d_ref, scale, accumulate, d_loss, d_adj_x);
    GS_CUDA(cudaGetLastError(), "k_loss_pos");
    count_launch();
    return GS_OK;
}

// centroid-trajectory loss over the frames of a rollout (SURVEY.md 8(b) gs_loss_centroid_traj_mse; BASELINE.json configs[3])
extern "C" int gs_loss_centroid_traj(gs_model *m, gs_tape *t, int frame_stride, const float *d_targets, float *d_loss, float *d_adj_x_frames,
                                     float *d_scratch_x, gs_stream stream) {
    GS_REQUIRE(m && t && t->m == m && d_targets && d_loss && d_scratch_x, GS_EINVAL, "null argument or foreign tape");
    GS_REQUIRE(t->has_rollout, GS_ESTATE, "the tape holds no rollout yet");
    GS_REQUIRE(frame_stride >= 1 && frame_stride <= t->T, GS_EINVAL, "frame_stride must be in [1, T]");
    GS_REQUIRE(t->K == 1 || frame_stride % t->K == 0, GS_EINVAL, "a checkpointed tape holds multiples of %d only", t->K);
    const int n_t = t->T / frame_stride;
    const size_t per = (size_t)m->E * m->N * 3;
    for (int f = 0; f < n_t; f++) {
        GS_TRY(gs_tape_read(m, t, (f + 1) * frame_stride, d_scratch_x, nullptr, stream));
        GS_TRY(gs_loss_centroid(m->E, m->N, d_scratch_x, d_targets + (size_t)f * m->E * 3, 1.0f / (float)n_t, f > 0, d_loss,
                                d_adj_x_frames ? d_adj_x_frames + (size_t)f * per : nullptr, stream));
    }
    return GS_OK;
}

// ------------------------------------------------------------------------------------------ host-buffer end-to-end
static size_t al256(size_t n) { return (n + 255) & ~(size_t)255; }

// loss times of a rollout of T substeps (SURVEY.md 8(c) "Losses"): the final state only, or every frame_stride-th
// substep (position loss: plus the final state when T is not a multiple)
static int loss_times(int kind, int T, int stride, int *n_frames, bool *final_extra) {
    *final_extra = false;
    if (kind == GS_LOSS_FINAL_CENTROID) { *n_frames = 0; return 1; }
    *n_frames = T / stride;
    *final_extra = kind == GS_LOSS_POS_FRAMES && T % stride != 0;
    return *n_frames + (*final_extra ? 1 : 0);
}
static size_t target_floats(const gs_model *m, int kind, int n_t) {
    const size_t per = kind == GS_LOSS_POS_FRAMES ? (size_t)m->E * m->N * 3 : (size_t)m->E * 3;
    return per * (size_t)n_t;
}

extern "C" size_t gs_host_scratch_bytes(const gs_model *m, const gs_tape *t, int loss_kind, int frame_stride) {
    if (!m || !t || loss_kind < GS_LOSS_FINAL_CENTROID || loss_kind > GS_LOSS_CENTROID_TRAJ || (loss_kind != GS_LOSS_FINAL_CENTROID && frame_stride < 1)) return 0;
    const size_t st = al256((size_t)m->E * m->N * 3 * sizeof(float));
    int cmax = m->N > 3 ? m->N : 3;  // gravity gradients are 3 per environment
    for (int k = 0; k < N_TYPES; k++) cmax = cmax > m->counts[k] ? cmax : m->counts[k];
    int n_frames = 0;
    bool extra = false;
    const int n_t = loss_times(loss_kind, t->T, frame_stride, &n_frames, &extra);
    return 6 * st + (size_t)n_frames * st + al256(target_floats(m, loss_kind, n_t) * sizeof(float)) + al256((size_t)m->E * sizeof(float)) +
           al256((size_t)m->E * cmax * sizeof(float)) + 256;
}

extern "C" int gs_rollout_loss_backward_host(gs_model *m, gs_tape *t, const float *h_x0, const float *h_v0, int loss_kind, int frame_stride,
                                             const float *h_target, float *h_loss, float *h_adj_x0, float *h_adj_v0, int n_groups, const int *groups,
                                             float *const *h_grads, void *d_scratch, size_t scratch_bytes, gs_stream stream) {
    GS_REQUIRE(m && t && h_x0 && h_v0 && h_target && d_scratch, GS_EINVAL, "null argument");
    GS_REQUIRE(t->m == m, GS_EINVAL, "tape belongs to another model");
    GS_REQUIRE(n_groups >= 0 && (n_groups == 0 || (groups && h_grads)), GS_EINVAL, "bad groups");
    GS_REQUIRE(loss_kind >= GS_LOSS_FINAL_CENTROID && loss_kind <= GS_LOSS_CENTROID_TRAJ, GS_EINVAL, "unknown loss kind %d", loss_kind);
    GS_REQUIRE(loss_kind == GS_LOSS_FINAL_CENTROID || (frame_stride >= 1 && frame_stride <= t->T), GS_EINVAL, "frame_stride must be in [1, T]");
    GS_REQUIRE(loss_kind == GS_LOSS_FINAL_CENTROID || t->K == 1 || frame_stride % t->K == 0, GS_EINVAL,
               "a checkpointed tape holds multiples of %d only: frame_stride %d is not one", t->K, frame_stride);
    const size_t need = gs_host_scratch_bytes(m, t, loss_kind, frame_stride);
    GS_REQUIRE(scratch_bytes >= need && ((uintptr_t)d_scratch & 255) == 0, GS_EINVAL, "scratch too small (%zu < %zu) or misaligned", scratch_bytes, need);
    cudaStream_t st = (cudaStream_t)stream;
    const int E = m->E, N = m->N, T = t->T;
    int n_frames = 0;
    bool extra = false;
    const int n_t = loss_times(loss_kind, T, frame_stride, &n_frames, &extra);
    const size_t sb = (size_t)E * N * 3 * sizeof(float), sa = al256(sb), tf = target_floats(m, loss_kind, n_t);
    char *p = (char *)d_scratch;
    float *d_x0 = (float *)p, *d_v0 = (float *)(p + sa), *d_xt = (float *)(p + 2 * sa), *d_cot = (float *)(p + 3 * sa);
    float *d_ax0 = (float *)(p + 4 * sa), *d_av0 = (float *)(p + 5 * sa);
    float *d_frames = (float *)(p + 6 * sa);  // [n_frames][E][N][3] cotangents of the frame states (sb bytes each, packed)
    float *d_tgt = (float *)(p + 6 * sa + al256((size_t)n_frames * sb));
    float *d_loss = (float *)((char *)d_tgt + al256(tf * sizeof(float)));
    float *d_g = (float *)((char *)d_loss + al256((size_t)E * sizeof(float)));
    GS_CUDA(cudaMemcpyAsync(d_x0, h_x0, sb, cudaMemcpyHostToDevice, st), "H2D x0");
    GS_CUDA(cudaMemcpyAsync(d_v0, h_v0, sb, cudaMemcpyHostToDevice, st), "H2D v0");
    GS_CUDA(cudaMemcpyAsync(d_tgt, h_target, tf * sizeof(float), cudaMemcpyHostToDevice, st), "H2D target");
    GS_TRY(gs_zero_grads(m, stream));
    GS_TRY(gs_rollout(m, t, d_x0, d_v0, d_xt, nullptr, stream));
    const float *cot_T = nullptr;
    if (loss_kind == GS_LOSS_FINAL_CENTROID) {
        GS_TRY(gs_loss_centroid(E, N, d_xt, d_tgt, 1.0f, 0, d_loss, d_cot, stream));
        cot_T = d_cot;
    } else {
        // L = 1/(n_t N) sum_f sum_i |x_i(t_f) - ref|^2   or   L = 1/n_t sum_f |c(t_f) - c*_f|^2; frame f = state after (f+1) stride
        const float scale = loss_kind == GS_LOSS_POS_FRAMES ? 1.0f / ((float)n_t * (float)N) : 1.0f / (float)n_t;
        const size_t per = tf / (size_t)n_t;
        for (int f = 0; f < n_t; f++) {
            const int ts = f < n_frames ? (f + 1) * frame_stride : T;  // f == n_frames: the extra final-state term
            float *cot = f < n_frames ? d_frames + (size_t)f * (sb / sizeof(float)) : d_cot;
            GS_TRY(gs_tape_read(m, t, ts, d_xt, nullptr, stream));
            if (loss_kind == GS_LOSS_POS_FRAMES) GS_TRY(gs_loss_pos(E, N, d_xt, d_tgt + (size_t)f * per, scale, f > 0, d_loss, cot, stream));
            else GS_TRY(gs_loss_centroid(E, N, d_xt, d_tgt + (size_t)f * per, scale, f > 0, d_loss, cot, stream));
            if (f >= n_frames) cot_T = d_cot;
        }
    }
    GS_TRY(gs_rollout_backward(m, t, n_frames, n_frames ? frame_stride : 1, n_frames ? d_frames : nullptr, cot_T, nullptr, d_ax0, d_av0, stream));
    if (h_loss) GS_CUDA(cudaMemcpyAsync(h_loss, d_loss, (size_t)E * sizeof(float), cudaMemcpyDeviceToHost, st), "D2H loss");
    if (h_adj_x0) GS_CUDA(cudaMemcpyAsync(h_adj_x0, d_ax0, sb, cudaMemcpyDeviceToHost, st), "D2H adj_x0");
    if (h_adj_v0) GS_CUDA(cudaMemcpyAsync(h_adj_v0, d_av0, sb, cudaMemcpyDeviceToHost, st), "D2H adj_v0");
    for (int k = 0; k < n_groups; k++) {
        const int g = groups[k];
        GS_REQUIRE(g >= 0 && g < GS_NUM_GROUPS && h_grads[k], GS_EINVAL, "bad group %d", g);
        const int c = g == GS_MASS ? N : (g == GS_GRAVITY ? 3 : (g == GS_HINGE_THETA0 || g == GS_HINGE_KB ? m->counts[T_HINGE] : (g >= GS_CONTACT_KE ? 1 : m->counts[g / 3])));
        GS_REQUIRE(g != GS_WIND, GS_EINVAL, "the wind has no gradient");
        if (c == 0) continue;
        GS_TRY(gs_param_grads(m, g, d_g, stream));
        // the staging buffer is reused: the copy is ordered before the next group's kernel on the same stream
        GS_CUDA(cudaMemcpyAsync(h_grads[k], d_g, (size_t)E * c * sizeof(float), cudaMemcpyDeviceToHost, st), "D2H grads");
    }
    GS_CUDA(cudaStreamSynchronize(st), "synchronize");
    int bad = -1;
    return gs_check_finite(m, stream, &bad);
}

// ------------------------------------------------------------------------------------------ kernel timing
gs_model::~gs_model() {
    gs::resident_release(this);
    for (cudaEvent_t e : ev_pool) cudaEventDestroy(e);
}
namespace gs {
static cudaEvent_t next_event(gs_model *m) {
    if (m->ev_used == m->ev_pool.size()) {
        cudaEvent_t e = nullptr;
        if (cudaEventCreate(&e) != cudaSuccess) return nullptr;
        m->ev_pool.push_back(e);
    }
    return m->ev_pool[m->ev_used++];
}
cudaEvent_t timing_begin(gs_model *m, cudaStream_t st) {
    cudaEvent_t a = next_event(m);
    if (a) cudaEventRecord(a, st);
    return a;
}
void timing_end(gs_model *m, int id, cudaEvent_t a, cudaStream_t st) {
    cudaEvent_t b = next_event(m);
    if (!b) return;
    cudaEventRecord(b, st);
    m->timed.push_back({id, a, b});
}
}  // namespace gs

extern "C" int gs_kernel_timing(gs_model *m, int enable) {
    GS_REQUIRE(m, GS_EINVAL, "model is null");
    m->timing = enable != 0;
    return GS_OK;
}
extern "C" int gs_kernel_times(gs_model *m, gs_stream stream, int n, double *ms_total, uint64_t *launches) {
    GS_REQUIRE(m && ms_total && launches && n >= GS_K_COUNT, GS_EINVAL, "bad argument");
    GS_CUDA(cudaStreamSynchronize((cudaStream_t)stream), "synchronize");
    for (int k = 0; k < n; k++) { ms_total[k] = 0.0; launches[k] = 0; }
    for (const gs_model::TimedLaunch &t : m->timed) {
        float ms = 0.f;
        GS_CUDA(cudaEventElapsedTime(&ms, t.a, t.b), "cudaEventElapsedTime");
        ms_total[t.id] += ms;
        launches[t.id]++;
    }
    m->timed.clear();
    m->ev_used = 0;
    return GS_OK;
}

extern "C" uint64_t gs_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }
extern "C" const char *gs_version(void) { return "gradsim-b200 0.1 (sm_100a)"; }
