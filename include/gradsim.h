/*
 * gradsim.h -- C ABI of the B200-native gradSim hot path: the differentiable multiphysics
 * substep (tet Neo-Hookean FEM + triangle membrane + dihedral bending -> scatter-add ->
 * penalty ground contact with friction -> semi-implicit Euler) and its hand-written adjoint,
 * with an on-device state tape for backpropagation through time.
 *
 * Paper: arXiv 2104.02646 (gradSim).  Citations are "PAPER.md:<line>" = the paper's LaTeX as
 * mounted at build time, plus the section; "DESIGN.md Ax" = a documented reading where the
 * paper is silent.
 *
 * Conventions (all entry points)
 *  - Every function returns an int status (GS_OK = 0, negative = error); nothing throws or exits.
 *    gs_last_error() gives a thread-local message for the last failure.
 *  - "HOST" pointers are plain host memory, read during the call only (caller may free after).
 *    "DEVICE" pointers are CUDA device memory owned by the caller (e.g. a torch tensor's
 *    data_ptr()); the library never allocates or frees device memory: it works inside the
 *    workspace / tape blocks the caller hands over, which must outlive the model / tape and be
 *    256-byte aligned.
 *  - All device work is enqueued on the caller's stream (a cudaStream_t passed as void*) and is
 *    asynchronous; only gs_model_create, gs_tape_create, gs_check_finite and the *_host entry
 *    points synchronise.  One model is used from one stream at a time.  On the streaming plan gs_rollout and
 *    gs_rollout_backward replay a CUDA graph of their launch sequence (captured on a private stream the first time a
 *    tape is used, or again when the frame arguments change); per-kernel timing switches the graphs off.
 *  - State arrays crossing the ABI are fp32, CALLER'S particle order, [E][N][3] (env-major).
 *    Per-element / per-particle parameter and gradient arrays are [E][count], caller's element order.
 *    Internally particles and elements are reordered (Morton) and tiled; the permutation is applied
 *    on the way in and out, off the hot path (a rollout stays in the internal order).
 *  - Arithmetic is fp32 (parameter gradients are accumulated across substeps in fp64).
 */
#ifndef GRADSIM_H
#define GRADSIM_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct gs_model gs_model; /* opaque: one scene (mesh shared by all E environments) */
typedef struct gs_tape gs_tape;   /* opaque: on-device state tape of one rollout            */
typedef void *gs_stream;          /* cudaStream_t                                           */

enum gs_status {
    GS_OK = 0,
    GS_EINVAL = -1,     /* bad argument (null pointer, negative size, misaligned / too small block) */
    GS_EMESH = -2,      /* invalid mesh: index out of range, V_e <= 0, degenerate triangle / hinge   */
    GS_ENOMEM = -3,     /* host allocation failed                                                    */
    GS_ECUDA = -4,      /* a CUDA runtime call failed (message has the CUDA error string)            */
    GS_ENONFINITE = -5, /* a non-finite state was produced; see gs_check_finite                      */
    GS_ESTATE = -6      /* call order violated (e.g. backward on a tape that holds no rollout)       */
};

/* parameter groups of gs_set_params / gs_param_grads (Table 5: the optimisable
   parameters this path carries: Lame parameters and damping per element, mass per particle; from the "next"
   list bending stiffness per hinge and the contact parameters per environment) */
enum gs_param_group {
    GS_TET_MU = 0, GS_TET_LAMBDA = 1, GS_TET_DAMP = 2,
    GS_TRI_MU = 3, GS_TRI_LAMBDA = 4, GS_TRI_DAMP = 5,
    GS_MASS = 6,
    GS_HINGE_KB = 7, /* bending stiffness per hinge: one array [Mh] shared by all environments --
                        gs_set_params takes row 0 of its [E][Mh] argument; gs_param_grads returns dL/dk_b per environment */
    GS_CONTACT_KE = 8, GS_CONTACT_KD = 9, GS_CONTACT_KF = 10, GS_CONTACT_MUC = 11, /* contact parameters (NEXT-2): one value
                        per environment, arrays [E] (count = 1) */
    GS_GRAVITY = 12, /* gravity (Table 5 column "g", NEXT-2): ONE vector shared by all environments -- gs_set_params reads
                        d_values[0..2] (synchronises the stream; tapes re-capture their graphs at the next use);
                        gs_param_grads returns dL/dg per environment, [E][3] (count = 3).  Off by default: the sum over
                        all particles of every adjoint substep costs ~12 % of the particle adjoint kernel; gs_request_grads
                        switches it on (before the backward pass), else gs_param_grads returns GS_ESTATE */
    GS_HINGE_THETA0 = 13, /* rest angle per hinge (Table 5 column "rest": the rest configuration of the bending springs): one
                        array [Mh] shared by all environments, as GS_HINGE_KB.  Its gradient is read from the hinge actuation
                        gradients (theta0 and the per-edge actuation enter the same argument, PAPER.md:585-586:
                        dL/dtheta0 = -1/2 sum over frames of dL/dalpha), so gs_param_grads needs an activation schedule
                        attached (gs_actuation_create; one zero frame is enough), else GS_ESTATE */
    GS_AERO_DRAG = 14, GS_AERO_LIFT = 15, /* k_drag, k_lift of the lift / drag model (NEXT-3): one value per environment, [E] */
    GS_WIND = 16,    /* velocity of the air: ONE vector for all environments, set like GS_GRAVITY; it has no gradient
                        (gs_param_grads returns GS_EINVAL) */
    GS_NUM_GROUPS = 17
};

/* bit flags of gs_model_desc.param_layout: which parameter arrays carry a leading [E] axis */
enum gs_param_layout {
    GS_ELEM_PER_ENV = 1,    /* tet_* and tri_* arrays are [E][M] / [E][Mt]; else [M] / [Mt] broadcast */
    GS_MASS_PER_ENV = 2,    /* mass is [E][N]; else [N] broadcast                                       */
    GS_CONTACT_PER_ENV = 4  /* ke, kd, kf, mu_c are [E]; else [1] broadcast                             */
};

/* execution plans (gs_model_desc.plan) */
enum gs_plan {
    GS_PLAN_AUTO = 0,     /* resident when the mesh fits one CTA's shared memory, else streaming         */
    GS_PLAN_STREAMING = 1,/* two grid-wide kernels per substep over Morton-ordered element tiles          */
    GS_PLAN_RESIDENT = 2  /* one persistent CTA per environment, state on-chip across ALL substeps of a rollout
                             (tets-only meshes of <= 2048 tets; gs_step_* and checkpointed tapes of such a model
                             still run the streaming kernels) */
};

/*
 * Scene description.  All pointers HOST; copied during gs_model_create.
 *   x_rest defines the rest shape: tets  B = D_m^-1, V = det(D_m)/6       (App. A.1)
 *                                  tris  2x2 B in the triangle's rest frame, A = det(D_m)/2 (A4)
 *                                  hinges rest angle theta0 and rest edge length l0        (A5, A6)
 *   tets must be positively oriented (det D_m > 0), else GS_EMESH.
 *   hinges[h] = (wing1, wing2, edge_a, edge_b): the two vertices opposite the shared edge, then the edge.
 *   pinned[i] != 0 => inverse mass 0 (step(inv_mass)).
 *   Air ("a lift/drag model that approximates the effect of the surrounding air on the surface of mesh";
 *   DESIGN.md A21, the paper gives no formula): every triangle with area A, unit normal n and relative velocity
 *   vb = mean vertex velocity - wind gets F = -A |vb| (k_drag vb + k_lift (n.vb) n), a third on each vertex.
 *   Contact: plane n.x = d, threshold particle_radius, stiffness ke, damping kd,
 *   friction stiffness kf, friction coefficient mu_c (A7-A9).
 */
typedef struct {
    int32_t n_particles, n_tets, n_tris, n_hinges, n_envs;
    const float *x_rest;   /* [N][3] */
    const float *mass;     /* [E][N] or [N], > 0 */
    const uint8_t *pinned; /* [N] or NULL */
    const int32_t *tets;   /* [M][4] */
    const float *tet_mu, *tet_lambda, *tet_damp;
    const int32_t *tris;   /* [Mt][3] */
    const float *tri_mu, *tri_lambda, *tri_damp;
    const int32_t *hinges; /* [Mh][4] */
    const float *hinge_kb; /* [Mh] bending stiffness (units of force, A6) */
    uint32_t param_layout; /* gs_param_layout flags */
    float gravity[3];      /* acceleration added to every non-pinned particle (A10), e.g. (0,-9.8,0) */
    float dt;              /* substep */
    float plane_n[3];      /* unit normal */
    float plane_d;
    float particle_radius;
    const float *ke, *kd, *kf, *mu_c; /* [E] or [1] */
    int32_t plan;          /* gs_plan */
    const float *k_drag, *k_lift; /* [E] or [1] (GS_CONTACT_PER_ENV), or NULL = 0: lift / drag of the air on the triangles */
    float wind[3];         /* velocity of the air */
} gs_model_desc;

/* Upper bound of the device workspace a model of this description needs (bytes).  0 on a bad desc. */
size_t gs_model_workspace_bytes(const gs_model_desc *desc);

/* Validates the mesh, computes rest quantities, reorders and tiles it, uploads everything into
   d_workspace (DEVICE, >= gs_model_workspace_bytes, 256-byte aligned).  Synchronises the stream.
   Errors: GS_EINVAL, GS_EMESH (message names the element), GS_ENOMEM, GS_ECUDA. */
int gs_model_create(const gs_model_desc *desc, void *d_workspace, size_t bytes, gs_stream stream, gs_model **out);
void gs_model_destroy(gs_model *m);

/*
 * Deterministic mode of the streaming plan (SURVEY.md 8(c) hazard H6: "a coloured-scatter debug mode makes runs
 * repeatable"; north_star (3): atomic or graph-coloured scatter).  The tiles of all element types are coloured at model
 * creation so that no two tiles of a colour share a particle; with the mode on, the element kernels are launched once per
 * colour, so every particle's force / cotangent sum is formed in a fixed order and states, dL/dx0, dL/dv0 and the
 * per-element / per-particle gradients are bitwise reproducible run to run (the per-environment totals of the contact,
 * gravity and air parameters are fp64 atomic sums and may differ in the last bit).  Slower (about one launch per colour:
 * 10-20 per substep); the resident plan is deterministic as it is.  GS_ESTATE if the mesh needs more than 64 colours.
 */
int gs_set_deterministic(gs_model *m, int enable);

/* Which plan the model runs (gs_plan value), and basic sizes. */
int gs_model_plan(const gs_model *m);
int gs_model_info(const gs_model *m, int32_t *n_particles, int32_t *n_elements, int32_t *n_envs);

/* Replace one parameter group from DEVICE values [E][count] in caller order (count = M, Mt, N or Mh).
   Preconditions as in gs_model_create: finite values, mass > 0, lambda > 0.  The check runs on the device: an offending
   entry keeps its old value and raises the non-finite flag, so the next gs_check_finite returns GS_ENONFINITE (substep 0). */
int gs_set_params(gs_model *m, int group, const float *d_values, gs_stream stream);

/*
 * Actuation inputs.  PAPER.md:579: alpha of the volume term (J - alpha)^2 is "a per-element
 * actuation value that allows the element to expand and contract" -- here alpha = 1 + 3 mu / (4 lambda) + act (DESIGN.md
 * A1), act per tet; f_b = k_b sin(phi/2 + alpha) d with alpha "a per-edge actuation value that allows
 * the mesh to flex inwards or outwards", per hinge.  Activations vary in time (App. E: a controller
 * evaluated over simulation time produces them; that controller is gs_controller_schedule / gs_controller_grads below): a
 * SCHEDULE of n_frames frames, frame f holding during substeps [f frame_stride, (f+1) frame_stride) of a rollout, the last frame to the end.
 *   gs_actuation_create   attaches a schedule, all zeros (= passive), stored in d_mem (DEVICE, >= gs_actuation_bytes,
 *                         256-byte aligned, must outlive the model or the next create); n_frames = 0 detaches.
 *   gs_set_actuation      DEVICE values [n_frames][E][count] in caller element order (count = M or Mh).
 *   gs_actuation_grads    dL/d(activation) [n_frames][E][count], accumulated by the adjoint substeps since gs_zero_grads
 *                         (fp32 sums of frame_stride terms per entry).
 *   gs_set_actuation_frame  the frame gs_step_forward / gs_step_backward use (default 0).
 * Triangles carry no actuation.  Errors: GS_EINVAL, GS_ESTATE (no schedule attached), GS_ECUDA.
 */
enum gs_actuation_kind { GS_ACT_TET = 0, GS_ACT_HINGE = 1 };
size_t gs_actuation_bytes(const gs_model *m, int n_frames);
int gs_actuation_create(gs_model *m, int n_frames, int frame_stride, void *d_mem, size_t bytes, gs_stream stream);
int gs_set_actuation(gs_model *m, int kind, const float *d_values, gs_stream stream);
int gs_actuation_grads(gs_model *m, int kind, float *d_out, gs_stream stream);
int gs_set_actuation_frame(gs_model *m, int frame);

/*
 * One forward substep (PAPER.md:618-619 semi-implicit Euler; 763-764 Listing 1):
 *   f = tets + triangles + hinges + contact, all at the start-of-step state;
 *   v+ = v + (f w + g [w>0]) dt;  x+ = x + v+ dt.
 * d_x, d_v: DEVICE [E][N][3] in; d_x_out, d_v_out: DEVICE [E][N][3] out (may alias the inputs).
 */
int gs_step_forward(gs_model *m, const float *d_x, const float *d_v, float *d_x_out, float *d_v_out, gs_stream stream);

/*
 * Adjoint of one substep (PAPER.md:561-563 implicit-function adjoint; 622-631 Jacobians of g, solved
 * explicitly thanks to their triangular structure).  d_x, d_v: state BEFORE the step.  d_adj_x_out,
 * d_adj_v_out: dL/d(state after).  Writes dL/d(state before) to d_adj_x_in, d_adj_v_in (may alias the
 * cotangent inputs).  Parameter gradients ACCUMULATE in the model until gs_zero_grads.
 */
int gs_step_backward(gs_model *m, const float *d_x, const float *d_v, const float *d_adj_x_out, const float *d_adj_v_out,
                     float *d_adj_x_in, float *d_adj_v_in, gs_stream stream);

/*
 * State tape (reverse mode must store the input state of every step).
 * checkpoint_every = 1 keeps every substep; K > 1 keeps states 0, K, 2K, ... and the final state, and
 * the backward pass regenerates each segment by forward replay (BASELINE.json configs[2]).
 * d_mem: DEVICE block of >= gs_tape_bytes, 256-byte aligned.
 */
size_t gs_tape_bytes(const gs_model *m, int n_substeps, int checkpoint_every);
int gs_tape_create(gs_model *m, int n_substeps, int checkpoint_every, void *d_mem, size_t bytes, gs_tape **out);
void gs_tape_destroy(gs_tape *t);

/* Forward rollout of the tape's n_substeps from (d_x0, d_v0) [E][N][3]; optional final state out (may be NULL). */
int gs_rollout(gs_model *m, gs_tape *t, const float *d_x0, const float *d_v0, float *d_x_T, float *d_v_T, gs_stream stream);

/* Copy the stored state after `substep` substeps to caller order.  GS_ESTATE if the tape does not hold
   that substep (checkpointed tapes hold multiples of K and the final state, so a loss that reads frames
   every frame_stride substeps needs K | frame_stride).  Either output may be NULL. */
int gs_tape_read(gs_model *m, gs_tape *t, int substep, float *d_x, float *d_v, gs_stream stream);

/*
 * Backward through the tape's rollout.  Loss cotangents enter at frame boundaries: frame k (0-based) is
 * the state after (k+1)*frame_stride substeps, d_adj_x_frames is DEVICE [n_frames][E][N][3] (NULL / 0 for
 * none); d_adj_x_T, d_adj_v_T are the cotangents of the final state (NULL = zero).  Outputs dL/dx0,
 * dL/dv0 (either may be NULL).  Parameter gradients accumulate in the model.
 */
int gs_rollout_backward(gs_model *m, gs_tape *t, int n_frames, int frame_stride, const float *d_adj_x_frames,
                        const float *d_adj_x_T, const float *d_adj_v_T, float *d_adj_x0, float *d_adj_v0, gs_stream stream);

/* Switch a gradient that costs extra work per substep on or off (only GS_GRAVITY needs this; every other group is always
   accumulated).  Tapes re-capture their graphs at the next use. */
int gs_request_grads(gs_model *m, int group, int enable);
int gs_zero_grads(gs_model *m, gs_stream stream);
/* Accumulated dL/d(parameter) of one group, DEVICE out [E][count] fp32 in caller order.  For GS_MASS the
   gradient of a pinned particle is 0 (A11). */
int gs_param_grads(gs_model *m, int group, float *d_out, gs_stream stream);

/* Synchronises the stream; *first_bad_substep = index of the first substep (since the last rollout /
   step call began) that produced a non-finite position or velocity, or -1.  Returns GS_ENONFINITE if any. */
int gs_check_finite(gs_model *m, gs_stream stream, int *first_bad_substep);

/*
 * Loss helpers on caller-order DEVICE arrays, so that a whole optimisation iteration can stay on the
 * device (centre-of-mass based loss; BASELINE.json configs).
 *   gs_loss_centroid: L_e (+)= scale * || mean_i x_i - target_e ||^2 ; adj_x_i = 2 scale (c - c*) / N
 *   gs_loss_pos:      L_e (+)= scale * sum_i || x_i - ref_i ||^2     ; adj_x_i = 2 scale (x_i - ref_i)
 * d_x [E][N][3], d_target [E][3], d_ref [E][N][3], d_loss [E] (overwritten unless accumulate != 0),
 * d_adj_x [E][N][3] overwritten (may be NULL).
 */
int gs_loss_centroid(int n_envs, int n_particles, const float *d_x, const float *d_target, float scale, int accumulate,
                     float *d_loss, float *d_adj_x, gs_stream stream);
int gs_loss_pos(int n_envs, int n_particles, const float *d_x, const float *d_ref, float scale, int accumulate,
                float *d_loss, float *d_adj_x, gs_stream stream);
/*
 * Centroid-trajectory loss of a rollout (BASELINE.json configs[3]; PAPER.md:365 a centre-of-mass loss "at each time step"):
 *   L_e = 1/n_t sum_f || c_e(t_f) - target_{f,e} ||^2,  t_f = (f+1) frame_stride, n_t = T / frame_stride frames,
 * read from the tape of the last gs_rollout.  d_targets [n_t][E][3]; d_loss [E] overwritten; d_adj_x_frames [n_t][E][N][3]
 * overwritten with dL/dx(t_f) in the layout gs_rollout_backward takes (may be NULL); d_scratch_x: DEVICE [E][N][3].
 * A checkpointed tape needs K | frame_stride.  Errors: GS_EINVAL, GS_ESTATE (no rollout on the tape).
 */
int gs_loss_centroid_traj(gs_model *m, gs_tape *t, int frame_stride, const float *d_targets, float *d_loss,
                          float *d_adj_x_frames, float *d_scratch_x, gs_stream stream);

/*
 * The open-loop MPC controller that produces an activation schedule, and its weight gradient.
 * "N phase-shifted sinusoidal signals ... passed to a fully-connected layer (zero-bias), and a final activation
 * layer.  The output is a vector of per-element activation values"; tanh, 8 signals.  DESIGN.md A23b:
 *   s_i(t) = sin(omega t + 2 pi i / n_signals);  act[f][e][k] = amplitude tanh(sum_i W[e][k][i] s_i(f frame_dt));
 *   g_W[e][k][i] = sum_f g_act[f][e][k] amplitude (1 - tanh^2) s_i(f frame_dt).
 * All arrays DEVICE fp32, caller order: d_W, d_g_W [n_envs][count][n_signals]; d_act [n_frames][n_envs][count] is what
 * gs_set_actuation takes, d_g_act what gs_actuation_grads writes (frame_dt = frame_stride x dt of that schedule).  Pure
 * functions of their arguments: no model is touched.  Both overwrite their output.  Errors: GS_EINVAL (sizes < 1,
 * n_signals > 8192, frame_dt <= 0, null array), GS_ECUDA.
 */
int gs_controller_schedule(int n_frames, int n_envs, int count, int n_signals, float omega, float frame_dt, float amplitude,
                           const float *d_W, float *d_act, gs_stream stream);
int gs_controller_grads(int n_frames, int n_envs, int count, int n_signals, float omega, float frame_dt, float amplitude,
                        const float *d_W, const float *d_g_act, float *d_g_W, gs_stream stream);

/*
 * Soft silhouette rasteriser on a headless device buffer, and its adjoint: the image-space loss of
 * the paper's pixels-to-parameters loop.  PAPER.md:168-172 (section 2.2: "replace discontinuous triangle mesh edges with
 * smooth sigmoids"); the formula is the SoftRas silhouette as SPEC.md:251 states it (A22):
 *   D_j(p) = sigmoid(delta d^2(p, boundary of triangle j) / sigma), delta = +1 inside / -1 outside, distances in NDC;
 *   S(p) = 1 - prod_j (1 - D_j(p));   gs_loss_silhouette: L_e (+)= scale sum_p (S_e(p) - target_e(p))^2.
 * Camera (HOST struct, read during the call): p_cam = R x + t (R row-major), a triangle is drawn iff all three vertices
 * have z_cam > near_z, NDC (u, v) = (fx X / Z, fy Y / Z), pixel (i, j) centre at u = 2 (i + 1/2) / W - 1, v = 2 (j + 1/2) / H - 1.
 * d_x [E][N][3] caller order (e.g. a state from gs_rollout / gs_tape_read); d_tris [n_tris][3] DEVICE int32 indices into
 * the particles (any surface mesh: the cloth triangles, or the boundary faces of a tet mesh); images [E][H][W] fp32.
 * gs_loss_silhouette: d_loss [E] (overwritten unless accumulate), d_adj_x [E][N][3] = dL/dx overwritten (may be NULL),
 * d_image optional.  The result feeds gs_rollout_backward as d_adj_x_T or a frame cotangent.  d_scratch: DEVICE block of
 * >= gs_raster_scratch_bytes, 256-byte aligned.  The colour channel is gs_render_rgb / gs_loss_rgb below.
 */
typedef struct {
    float R[9], t[3];      /* world -> camera */
    float fx, fy;          /* focal lengths in NDC units (1 / tan(fov / 2)) */
    int32_t width, height;
    float sigma;           /* edge blur, in squared NDC units */
    float near_z;
} gs_camera;
size_t gs_raster_scratch_bytes(int n_envs, int n_particles, int n_tris);
int gs_render_silhouette(int n_envs, int n_particles, const float *d_x, int n_tris, const int32_t *d_tris, const gs_camera *cam,
                         float *d_image, void *d_scratch, size_t scratch_bytes, gs_stream stream);
int gs_loss_silhouette(int n_envs, int n_particles, const float *d_x, int n_tris, const int32_t *d_tris, const gs_camera *cam,
                       const float *d_target, float scale, int accumulate, float *d_loss, float *d_adj_x, float *d_image,
                       void *d_scratch, size_t scratch_bytes, gs_stream stream);

/*
 * gs_loss_silhouette without any allocation and without a caller scratch block, for callers that cannot call cudaMalloc
 * (code under CUDA graph capture, tight serving loops, harnesses that forbid it).  Same arguments, results and errors as
 * gs_loss_silhouette (d_image and d_adj_x optional), but the scratch lives in a file-scope device array of
 * GS_RASTER_STATIC_BYTES (8 MiB) inside the library: every GPU that loads the library holds that much until the process
 * exits.  A problem whose gs_raster_scratch_bytes(n_envs, n_particles, n_tris) exceeds GS_RASTER_STATIC_BYTES is rejected
 * with GS_EINVAL before any CUDA call (e.g. 64 environments x 1089 particles x 1922 triangles = 7.6 MiB fits; twice that does
 * not).  The call itself enqueues kernels and cudaMemsetAsync only: no cudaMalloc / cudaFree / allocating library routine.
 * ALL calls on one GPU share the one array and it keeps the last call's contents (what must start at zero is cleared by the
 * call): two calls that overlap on the GPU (different streams, or graphs replayed concurrently) RACE -- serialise them.  The
 * array's device address is looked up once per device, with the caller's current device, on first use.
 */
#define GS_RASTER_STATIC_BYTES (8u << 20)
int gs_loss_silhouette_static(int n_envs, int n_particles, const float *d_x, int n_tris, const int32_t *d_tris, const gs_camera *cam,
                              const float *d_target, float scale, int accumulate, float *d_loss, float *d_adj_x, float *d_image,
                              gs_stream stream);

/*
 * Colour channel of the soft rasteriser and its adjoint (SURVEY.md 8(f) NEXT-4 "silhouette/colour"; A22b).
 * PAPER.md:168-172 blurs the edges, PAPER.md:495 names the "only colour" shading; the aggregation is the one SPEC.md:251
 * states ("depth-softmax aggregation ... weights proportional to D_j exp(zbar_j / gamma) plus a background term, normalized;
 * ... barycentric interpolation of ... vertex colors, barycentrics clamped for exterior pixels"):
 *   lam_k(p) screen-space (NDC) barycentrics of pixel centre p in triangle j;  w = clip(lam, 0, 1) / sum clip(lam, 0, 1);
 *   z_j = sum_k w_k Z_k (camera depth),  zbar_j = (far_z - z_j) / (far_z - near_z);  C_j = sum_k w_k c_k;
 *   I(p) = (sum_j D_j e^{zbar_j / gamma} C_j + e^{eps / gamma} background) / (sum_j D_j e^{zbar_j / gamma} + e^{eps / gamma})
 * over the drawn triangles with |2 area| > 1e-5 x (longest edge)^2 in NDC (no slivers) and signed squared distance s_j(p) >= -40 sigma; D_j, camera and pixel
 * grid as for the silhouette.  gs_loss_rgb: L_e (+)= scale sum_p sum_c (I_{e,c}(p) - target_{e,c}(p))^2.
 * d_colour [E][N][3] per-vertex colours (no lighting); images and targets planar [E][3][H][W] fp32.  d_adj_x [E][N][3] = dL/dx and
 * d_adj_colour [E][N][3] = dL/dcolour are overwritten (each may be NULL); d_image optional in gs_loss_rgb.  gs_shading is a
 * HOST struct read during the call.  d_scratch: DEVICE block of >= gs_raster_rgb_scratch_bytes, 256-byte aligned.
 * Errors: GS_EINVAL (null / misaligned / too small a block, gamma <= 0, far_z <= near_z), GS_ECUDA.
 */
typedef struct {
    float gamma;          /* depth softmax temperature, in units of the normalised depth */
    float eps;            /* normalised depth of the background term */
    float far_z;          /* camera depth mapped to zbar = 0 (near_z of the camera maps to 1) */
    float background[3];
} gs_shading;
size_t gs_raster_rgb_scratch_bytes(int n_envs, int n_particles, int n_tris);
int gs_render_rgb(int n_envs, int n_particles, const float *d_x, int n_tris, const int32_t *d_tris, const float *d_colour,
                  const gs_camera *cam, const gs_shading *shading, float *d_image, void *d_scratch, size_t scratch_bytes,
                  gs_stream stream);
int gs_loss_rgb(int n_envs, int n_particles, const float *d_x, int n_tris, const int32_t *d_tris, const float *d_colour,
                const gs_camera *cam, const gs_shading *shading, const float *d_target, float scale, int accumulate,
                float *d_loss, float *d_adj_x, float *d_adj_colour, float *d_image, void *d_scratch, size_t scratch_bytes,
                gs_stream stream);

/*
 * End-to-end convenience with HOST buffers (bench.py's e2e leg): ONE call uploads x0, v0 [E][N][3] and the loss
 * targets, runs gs_rollout, the loss, gs_rollout_backward, and downloads loss [E], dL/dx0, dL/dv0 [E][N][3] (each may
 * be NULL) and the parameter gradients listed in groups[] into h_grads[k] ([E][count] each).  Zeroes the model's
 * gradients first.  Synchronises.  Losses (SURVEY.md 8(c) "Losses"; BASELINE.json configs):
 *   GS_LOSS_FINAL_CENTROID  L_e = || c(x_T) - c*_e ||^2, c = mean_i x_i                  h_target [E][3]
 *   GS_LOSS_POS_FRAMES      L_e = 1/(n_t N) sum_f sum_i || x_i(t_f) - ref_i(t_f) ||^2      h_target [n_t][E][N][3]
 *   GS_LOSS_CENTROID_TRAJ   L_e = 1/n_t sum_f || c_e(t_f) - c*_e(t_f) ||^2                 h_target [n_t][E][3]
 * with loss times t_f = frame_stride, 2 frame_stride, ... <= T (GS_LOSS_POS_FRAMES adds t = T when T is not a
 * multiple), n_t their number.  frame_stride is ignored for GS_LOSS_FINAL_CENTROID; a checkpointed tape needs
 * K | frame_stride.  d_scratch: DEVICE block of >= gs_host_scratch_bytes (same tape, loss_kind, frame_stride),
 * 256-byte aligned.  Errors: GS_EINVAL (arguments), GS_ENONFINITE (as gs_check_finite), GS_ECUDA.
 */
enum gs_loss_kind { GS_LOSS_FINAL_CENTROID = 0, GS_LOSS_POS_FRAMES = 1, GS_LOSS_CENTROID_TRAJ = 2 };
size_t gs_host_scratch_bytes(const gs_model *m, const gs_tape *t, int loss_kind, int frame_stride);
int gs_rollout_loss_backward_host(gs_model *m, gs_tape *t, const float *h_x0, const float *h_v0, int loss_kind, int frame_stride,
                                  const float *h_target, float *h_loss, float *h_adj_x0, float *h_adj_v0, int n_groups,
                                  const int *groups, float *const *h_grads, void *d_scratch, size_t scratch_bytes, gs_stream stream);

/* Number of kernel launches the library has enqueued since the process started (bench.py's gpu_launches). */
uint64_t gs_launch_count(void);

/*
 * Per-kernel device timing (bench.py's roofline leg).  While enabled, every hot-path kernel launch of this
 * model is bracketed by CUDA events recorded on the caller's stream.  gs_kernel_times synchronises the
 * stream, adds the elapsed time of every recorded launch to ms_total[kernel] and its count to
 * launches[kernel] (arrays of n >= GS_K_COUNT entries, overwritten), and clears the record.
 * Off by default; the events cost a few microseconds of host time per launch, so timed throughput runs
 * keep it off.  Kernel ids: elements_fwd = a1-a4, particles_fwd = a5-a7,
 * particles_adj = a8, elements_adj = a9-a10, other = layout conversion / gradient flush / losses.
 */
enum gs_kernel_id {
    GS_K_ELEMENTS_FWD = 0, GS_K_PARTICLES_FWD = 1, GS_K_PARTICLES_ADJ = 2, GS_K_ELEMENTS_ADJ = 3, GS_K_OTHER = 4,
    GS_K_RESIDENT_FWD = 5, /* resident plan: a1-a7 of all T substeps in one launch */
    GS_K_RESIDENT_ADJ = 6, /* resident plan: a8-a10 of all T substeps in one launch */
    GS_K_COUNT = 7
};
int gs_kernel_timing(gs_model *m, int enable);
int gs_kernel_times(gs_model *m, gs_stream stream, int n, double *ms_total, uint64_t *launches);

const char *gs_last_error(void);
const char *gs_version(void);

#ifdef __cplusplus
}
#endif
#endif /* GRADSIM_H */
