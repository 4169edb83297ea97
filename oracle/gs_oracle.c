/*
 * gs_oracle.c -- fp64 CPU oracle of the gradSim differentiable multiphysics substep
 * and its reverse-mode adjoint.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code,
 * header, table or helper with the CUDA path in paper_2104_02646_b200/csrc.
 *
 * Plain C99, plain loops, AoS doubles, one element at a time, in the paper's order and
 * notation.  Forces are accumulated per particle in a fixed order (tets, triangles,
 * hinges in increasing element index, then contact), so results are deterministic and
 * independent of the OpenMP thread count (OpenMP only splits independent loop
 * iterations: environments, elements writing private slots, particles gathering).
 *
 * What each function follows (PAPER.md = /root/reference/PAPER.md, the paper's LaTeX):
 *   tet_force / tet_energy      PAPER.md:575-581 (App. A.1 "Deformable Solids", Psi, U, f=-grad U),
 *                               PAPER.md:659-665 (App. C.1); readings A1 (alpha), A3 (damping)
 *   tri_force / tri_energy      PAPER.md:584 ("Deformable Thin-Shells": same Psi in-plane); reading A4
 *   hinge_force / hinge_energy  PAPER.md:585-586 (f_b = k_b sin(phi/2+alpha) d); readings A5, A6
 *   contact_force               PAPER.md:596-599, 684-688 (compliant contact, relaxed Coulomb); A7, A8
 *   integrate                   PAPER.md:618-619 (semi-implicit Euler g(s-,s+,theta)=0), 763-764 (Listing 1); A10, A11
 *   *_adjoint, step_adjoint     PAPER.md:561-563 (implicit-function adjoint), 622-631 (Jacobians of g;
 *                               "triangular structure ... computed explicitly")
 *   rollout, rollout_backward   PAPER.md:613 (reverse mode stores the input state of every step);
 *                               checkpoint + replay per BASELINE.json configs[2]
 *   aero_force / aero_adjoint   PAPER.md:586 (lift / drag of the air on the cloth faces); reading A21
 *   actuation inputs            PAPER.md:579 (per-tet alpha of (J - alpha)^2), 585-586 (per-edge alpha of sin(phi/2 + alpha)),
 *                               777 (App. E: activations produced in time by a controller); SURVEY.md 8(f) NEXT-1
 * Readings A1..A20 are listed in DESIGN.md ("Readings of the paper").
 *
 * Pins (tests/test_oracle_pins.py): P1..P10 of DESIGN.md.  Unpinned: the CHOICE among
 * alternative readings A3, A4, A6, A7, A8, A9 (the paper does not decide them) -- "parity
 * unpinned" for that choice only; every formula below is pinned for the reading taken.
 */
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

typedef struct {
    int N, M, Mt, Mh, E;
    double *mass;          /* [E][N] */
    unsigned char *pinned; /* [N] */
    int *tets;             /* [M][4] */
    double *tet_B;         /* [M][9] row-major inverse rest edge matrix D_m^-1 */
    double *tet_V;         /* [M] rest volume */
    double *tet_mu, *tet_lambda, *tet_damp; /* [E][M] */
    int *tris;             /* [Mt][3] */
    double *tri_B;         /* [Mt][4] row-major 2x2 */
    double *tri_A;         /* [Mt] rest area */
    double *tri_mu, *tri_lambda, *tri_damp; /* [E][Mt] */
    int *hinges;           /* [Mh][4] = wing1, wing2, edge_a, edge_b */
    double *hinge_theta0, *hinge_l0, *hinge_kb; /* [Mh] */
    double g[3], dt, n[3], d, r;
    double *ke, *kd, *kf, *mu_c; /* [E] */
    /* lift / drag of the surrounding air on the cloth triangles ("We also include a lift/drag model that
       approximates the effect of the surrounding air on the surface of mesh"; reading A21: the paper gives no formula) */
    double *k_drag, *k_lift;     /* [E], 0 = none */
    double wind[3];              /* velocity of the air */
    double *g_kdrag, *g_klift;   /* [E] dL/dk_drag, dL/dk_lift */
    /* incident lists: for particle i, entries inc_ptr[i]..inc_ptr[i+1] of inc_slot index
       the per-element-vertex slot arrays (tets: 4 slots, then tris: 3, then hinges: 4) */
    int *inc_ptr, *inc_slot;
    int n_slots;
    /* parameter-gradient accumulators (sum over substeps) */
    double *g_tet_mu, *g_tet_lambda, *g_tet_damp; /* [E][M] */
    double *g_tri_mu, *g_tri_lambda, *g_tri_damp; /* [E][Mt] */
    double *g_mass;                               /* [E][N] */
    double *g_ke, *g_kd, *g_kf, *g_muc;           /* [E]  dL/d(contact parameters) per environment (Table 5: contact parameters are optimisable) */
    double *g_hinge_kb;                           /* [E][Mh]  dL/dk_b per hinge (Table 5: bending stiffness is optimisable) */
    double *g_gravity;                            /* [E][3]   dL/dg per environment (Table 5 column "g") */
    /* actuation ("alpha is a per-element actuation value that allows the element to expand and contract";
       585-586 "alpha is a per-edge actuation value that allows the mesh to flex inwards or outwards"): CURRENT values used by
       orc_step / orc_step_adjoint, and their per-substep gradients.  Rollouts copy one frame of the schedule in before every
       substep (piecewise-constant control, one frame per act_stride substeps: App. E, a controller evaluated
       in time) and add the substep's gradient to that frame's slot. */
    double *tet_act, *hinge_act;                  /* [E][M], [E][Mh]; zero = passive */
    double *g_tet_act, *g_hinge_act;              /* [E][M], [E][Mh] dL/d(act) of the substeps since they were last cleared */
    int act_frames, act_stride;                   /* schedule: frame f holds for substeps [f stride, (f+1) stride); 0 frames = none */
    double *sched_tet, *sched_hinge;              /* [F][E][M], [F][E][Mh] (NULL = that kind is not actuated) */
    double *g_sched_tet, *g_sched_hinge;          /* gradients of the schedule, same shapes */
    double *g_hinge_theta0;                       /* [E][Mh] dL/d(rest angle) (Table 5 column "rest": the rest configuration of the bending springs) */
    double *g_con_abs;                            /* [E][4]   diagnostic only: sum of |term| behind g_ke, g_kd, g_kf, g_muc (how far each total cancels) */
} orc_model;

static char g_err[256] = "";
const char *orc_last_error(void) { return g_err; }

/* ---------------------------------------------------------------- small vector helpers */
static void v_sub(const double *a, const double *b, double *o) { o[0] = a[0] - b[0]; o[1] = a[1] - b[1]; o[2] = a[2] - b[2]; }
static double v_dot(const double *a, const double *b) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }
static void v_cross(const double *a, const double *b, double *o) {
    double x = a[1] * b[2] - a[2] * b[1], y = a[2] * b[0] - a[0] * b[2], z = a[0] * b[1] - a[1] * b[0];
    o[0] = x; o[1] = y; o[2] = z;
}
static void v_axpy(double s, const double *a, double *o) { o[0] += s * a[0]; o[1] += s * a[1]; o[2] += s * a[2]; }
static void v_scale(double s, const double *a, double *o) { o[0] = s * a[0]; o[1] = s * a[1]; o[2] = s * a[2]; }

/* 3x3 row-major helpers; column k of A is (A[k], A[3+k], A[6+k]) */
static void m_mul(const double *A, const double *B, double *C) { /* C = A B */
    double T[9];
    for (int r = 0; r < 3; r++) for (int c = 0; c < 3; c++) T[r * 3 + c] = A[r * 3] * B[c] + A[r * 3 + 1] * B[3 + c] + A[r * 3 + 2] * B[6 + c];
    memcpy(C, T, sizeof T);
}
static void m_mul_nt(const double *A, const double *B, double *C) { /* C = A B^T */
    double T[9];
    for (int r = 0; r < 3; r++) for (int c = 0; c < 3; c++) T[r * 3 + c] = A[r * 3] * B[c * 3] + A[r * 3 + 1] * B[c * 3 + 1] + A[r * 3 + 2] * B[c * 3 + 2];
    memcpy(C, T, sizeof T);
}
static void m_mul_tn(const double *A, const double *B, double *C) { /* C = A^T B */
    double T[9];
    for (int r = 0; r < 3; r++) for (int c = 0; c < 3; c++) T[r * 3 + c] = A[r] * B[c] + A[3 + r] * B[3 + c] + A[6 + r] * B[6 + c];
    memcpy(C, T, sizeof T);
}
static double m_ddot(const double *A, const double *B) { double s = 0; for (int i = 0; i < 9; i++) s += A[i] * B[i]; return s; }
static double m_det(const double *A) {
    return A[0] * (A[4] * A[8] - A[5] * A[7]) - A[1] * (A[3] * A[8] - A[5] * A[6]) + A[2] * (A[3] * A[7] - A[4] * A[6]);
}
static void m_col(const double *A, int k, double *c) { c[0] = A[k]; c[1] = A[3 + k]; c[2] = A[6 + k]; }
static void m_setcol(double *A, int k, const double *c) { A[k] = c[0]; A[3 + k] = c[1]; A[6 + k] = c[2]; }
static void m_sym(const double *A, double *S) { /* S = (A + A^T)/2 */
    double T[9];
    for (int r = 0; r < 3; r++) for (int c = 0; c < 3; c++) T[r * 3 + c] = 0.5 * (A[r * 3 + c] + A[c * 3 + r]);
    memcpy(S, T, sizeof T);
}
/* cof F = [f2 x f3, f3 x f1, f1 x f2] (columns) = dJ/dF, J = det F */
static void m_cof(const double *F, double *C) {
    double f1[3], f2[3], f3[3], c[3];
    m_col(F, 0, f1); m_col(F, 1, f2); m_col(F, 2, f3);
    v_cross(f2, f3, c); m_setcol(C, 0, c);
    v_cross(f3, f1, c); m_setcol(C, 1, c);
    v_cross(f1, f2, c); m_setcol(C, 2, c);
}
/* directional derivative of cof F along A: [a2 x f3 + f2 x a3, a3 x f1 + f3 x a1, a1 x f2 + f1 x a2] */
static void m_dcof(const double *F, const double *A, double *D) {
    double f[3][3], a[3][3], c1[3], c2[3];
    for (int k = 0; k < 3; k++) { m_col(F, k, f[k]); m_col(A, k, a[k]); }
    for (int k = 0; k < 3; k++) {
        int p = (k + 1) % 3, q = (k + 2) % 3;
        v_cross(a[p], f[q], c1); v_cross(f[p], a[q], c2);
        c1[0] += c2[0]; c1[1] += c2[1]; c1[2] += c2[2];
        m_setcol(D, k, c1);
    }
}

/* ---------------------------------------------------------------- model */
void orc_destroy(orc_model *m) {
    if (!m) return;
    free(m->mass); free(m->pinned); free(m->tets); free(m->tet_B); free(m->tet_V);
    free(m->tet_mu); free(m->tet_lambda); free(m->tet_damp);
    free(m->tris); free(m->tri_B); free(m->tri_A); free(m->tri_mu); free(m->tri_lambda); free(m->tri_damp);
    free(m->hinges); free(m->hinge_theta0); free(m->hinge_l0); free(m->hinge_kb);
    free(m->ke); free(m->kd); free(m->kf); free(m->mu_c);
    free(m->inc_ptr); free(m->inc_slot);
    free(m->g_tet_mu); free(m->g_tet_lambda); free(m->g_tet_damp);
    free(m->g_tri_mu); free(m->g_tri_lambda); free(m->g_tri_damp); free(m->g_mass); free(m->g_hinge_kb); free(m->g_ke); free(m->g_kd); free(m->g_kf); free(m->g_muc);
    free(m->g_gravity); free(m->g_con_abs); free(m->k_drag); free(m->k_lift); free(m->g_kdrag); free(m->g_klift);
    free(m->tet_act); free(m->hinge_act); free(m->g_tet_act); free(m->g_hinge_act); free(m->sched_tet); free(m->sched_hinge);
    free(m->g_sched_tet); free(m->g_sched_hinge); free(m->g_hinge_theta0);
    free(m);
}

static double *dup_d(const double *s, size_t n) { double *p = (double *)malloc((n ? n : 1) * sizeof(double)); if (n) memcpy(p, s, n * sizeof(double)); return p; }
static int *dup_i(const int *s, size_t n) { int *p = (int *)malloc((n ? n : 1) * sizeof(int)); if (n) memcpy(p, s, n * sizeof(int)); return p; }
static double *zeros_d(size_t n) { return (double *)calloc(n ? n : 1, sizeof(double)); }

/* signed dihedral angle theta (0 when flat) of hinge vertices x1,x2 (wings), x3,x4 (edge);
   optionally the Bridson directions d[4][3] = -d(theta)/dx_i.  PAPER.md:585-586, reading A5. */
static double hinge_angle(const double *x1, const double *x2, const double *x3, const double *x4, double d[4][3]) {
    double p13[3], p14[3], p23[3], p24[3], n1[3], n2[3], e[3], eh[3], c[3];
    v_sub(x1, x3, p13); v_sub(x1, x4, p14); v_sub(x2, x3, p23); v_sub(x2, x4, p24);
    v_cross(p13, p14, n1); v_cross(p24, p23, n2); v_sub(x4, x3, e);
    double L = sqrt(v_dot(e, e)), n1s = v_dot(n1, n1), n2s = v_dot(n2, n2);
    v_scale(1.0 / L, e, eh);
    double nh1[3], nh2[3];
    v_scale(1.0 / sqrt(n1s), n1, nh1); v_scale(1.0 / sqrt(n2s), n2, nh2);
    v_cross(nh1, nh2, c);
    double theta = atan2(v_dot(c, eh), v_dot(nh1, nh2));
    if (d) {
        double m1[3], m2[3];
        v_scale(1.0 / n1s, n1, m1); v_scale(1.0 / n2s, n2, m2);
        v_scale(L, m1, d[0]);
        v_scale(L, m2, d[1]);
        v_scale(v_dot(p14, eh), m1, d[2]); v_axpy(v_dot(p24, eh), m2, d[2]);
        v_scale(-v_dot(p13, eh), m1, d[3]); v_axpy(-v_dot(p23, eh), m2, d[3]);
    }
    return theta;
}

/* All arrays are full-shape doubles ([E][N], [E][M], ...).  Returns NULL on an invalid mesh
   (message in orc_last_error): index out of range, non-positive tet volume, degenerate triangle. */
orc_model *orc_create(int N, int M, int Mt, int Mh, int E, const double *x_rest, const double *mass,
                      const unsigned char *pinned, const int *tets, const double *tet_mu, const double *tet_lambda,
                      const double *tet_damp, const int *tris, const double *tri_mu, const double *tri_lambda,
                      const double *tri_damp, const int *hinges, const double *hinge_kb, const double *gravity,
                      double dt, const double *plane_n, double plane_d, double radius, const double *ke,
                      const double *kd, const double *kf, const double *mu_c) {
    orc_model *m = (orc_model *)calloc(1, sizeof(orc_model));
    m->N = N; m->M = M; m->Mt = Mt; m->Mh = Mh; m->E = E;
    m->mass = dup_d(mass, (size_t)E * N);
    m->pinned = (unsigned char *)calloc(N ? N : 1, 1);
    if (pinned) memcpy(m->pinned, pinned, N);
    m->tets = dup_i(tets, (size_t)M * 4);
    m->tet_mu = dup_d(tet_mu, (size_t)E * M); m->tet_lambda = dup_d(tet_lambda, (size_t)E * M); m->tet_damp = dup_d(tet_damp, (size_t)E * M);
    m->tris = dup_i(tris, (size_t)Mt * 3);
    m->tri_mu = dup_d(tri_mu, (size_t)E * Mt); m->tri_lambda = dup_d(tri_lambda, (size_t)E * Mt); m->tri_damp = dup_d(tri_damp, (size_t)E * Mt);
    m->hinges = dup_i(hinges, (size_t)Mh * 4);
    m->hinge_kb = dup_d(hinge_kb, Mh);
    m->tet_B = zeros_d((size_t)M * 9); m->tet_V = zeros_d(M);
    m->tri_B = zeros_d((size_t)Mt * 4); m->tri_A = zeros_d(Mt);
    m->hinge_theta0 = zeros_d(Mh); m->hinge_l0 = zeros_d(Mh);
    for (int k = 0; k < 3; k++) { m->g[k] = gravity[k]; m->n[k] = plane_n[k]; }
    m->dt = dt; m->d = plane_d; m->r = radius;
    m->ke = dup_d(ke, E); m->kd = dup_d(kd, E); m->kf = dup_d(kf, E); m->mu_c = dup_d(mu_c, E);
    m->g_tet_mu = zeros_d((size_t)E * M); m->g_tet_lambda = zeros_d((size_t)E * M); m->g_tet_damp = zeros_d((size_t)E * M);
    m->g_tri_mu = zeros_d((size_t)E * Mt); m->g_tri_lambda = zeros_d((size_t)E * Mt); m->g_tri_damp = zeros_d((size_t)E * Mt);
    m->g_mass = zeros_d((size_t)E * N);
    m->g_hinge_kb = zeros_d((size_t)E * Mh);
    m->g_ke = zeros_d((size_t)E); m->g_kd = zeros_d((size_t)E); m->g_kf = zeros_d((size_t)E); m->g_muc = zeros_d((size_t)E);
    m->g_gravity = zeros_d((size_t)E * 3); m->g_con_abs = zeros_d((size_t)E * 4);
    m->k_drag = zeros_d(E); m->k_lift = zeros_d(E); m->g_kdrag = zeros_d(E); m->g_klift = zeros_d(E);
    m->tet_act = zeros_d((size_t)E * M); m->hinge_act = zeros_d((size_t)E * Mh);
    m->g_tet_act = zeros_d((size_t)E * M); m->g_hinge_act = zeros_d((size_t)E * Mh); m->g_hinge_theta0 = zeros_d((size_t)E * Mh);

    /* tets: D_m = [X1-X0, X2-X0, X3-X0] (columns), B = D_m^-1, V = det(D_m)/6  (V_e) */
    for (int e = 0; e < M; e++) {
        const int *t = tets + 4 * e;
        for (int k = 0; k < 4; k++) if (t[k] < 0 || t[k] >= N) { snprintf(g_err, sizeof g_err, "tet %d: index out of range", e); orc_destroy(m); return NULL; }
        double Dm[9], c[3];
        for (int k = 0; k < 3; k++) { v_sub(x_rest + 3 * t[k + 1], x_rest + 3 * t[0], c); m_setcol(Dm, k, c); }
        double det = m_det(Dm);
        if (!(det > 0)) { snprintf(g_err, sizeof g_err, "tet %d: non-positive rest volume", e); orc_destroy(m); return NULL; }
        double C[9]; m_cof(Dm, C); /* inverse = cof^T / det */
        double *B = m->tet_B + 9 * e;
        for (int r = 0; r < 3; r++) for (int cc = 0; cc < 3; cc++) B[r * 3 + cc] = C[cc * 3 + r] / det;
        m->tet_V[e] = det / 6.0;
    }
    /* triangles: rest frame t1, t2 in the triangle plane, 2x2 D_m, B = D_m^-1, A = det(D_m)/2 (reading A4) */
    for (int e = 0; e < Mt; e++) {
        const int *t = tris + 3 * e;
        for (int k = 0; k < 3; k++) if (t[k] < 0 || t[k] >= N) { snprintf(g_err, sizeof g_err, "triangle %d: index out of range", e); orc_destroy(m); return NULL; }
        double e1[3], e2[3], nn[3], t1[3], t2[3];
        v_sub(x_rest + 3 * t[1], x_rest + 3 * t[0], e1); v_sub(x_rest + 3 * t[2], x_rest + 3 * t[0], e2);
        v_cross(e1, e2, nn);
        double l1 = sqrt(v_dot(e1, e1)), ln = sqrt(v_dot(nn, nn));
        if (!(0.5 * ln > 1e-12) || !(l1 > 0)) { snprintf(g_err, sizeof g_err, "triangle %d: degenerate rest shape", e); orc_destroy(m); return NULL; }
        v_scale(1.0 / l1, e1, t1); v_scale(1.0 / ln, nn, nn); v_cross(nn, t1, t2);
        double a = v_dot(t1, e1), b = v_dot(t1, e2), c = v_dot(t2, e1), dd = v_dot(t2, e2); /* D_m = [[a,b],[c,dd]] */
        double det = a * dd - b * c;
        double *B = m->tri_B + 4 * e;
        B[0] = dd / det; B[1] = -b / det; B[2] = -c / det; B[3] = a / det;
        m->tri_A[e] = det / 2.0;
    }
    /* hinges: rest angle theta0 and rest edge length l0 (readings A5, A6) */
    for (int e = 0; e < Mh; e++) {
        const int *h = hinges + 4 * e;
        for (int k = 0; k < 4; k++) if (h[k] < 0 || h[k] >= N) { snprintf(g_err, sizeof g_err, "hinge %d: index out of range", e); orc_destroy(m); return NULL; }
        m->hinge_theta0[e] = hinge_angle(x_rest + 3 * h[0], x_rest + 3 * h[1], x_rest + 3 * h[2], x_rest + 3 * h[3], NULL);
        double ed[3]; v_sub(x_rest + 3 * h[3], x_rest + 3 * h[2], ed);
        m->hinge_l0[e] = sqrt(v_dot(ed, ed));
    }
    /* incident slot lists in fixed order: tets, then triangles, then hinges, increasing element index */
    m->n_slots = 4 * M + 3 * Mt + 4 * Mh;
    m->inc_ptr = (int *)calloc((size_t)N + 1, sizeof(int));
    m->inc_slot = (int *)malloc((m->n_slots ? m->n_slots : 1) * sizeof(int));
    for (int e = 0; e < M; e++) for (int k = 0; k < 4; k++) m->inc_ptr[tets[4 * e + k] + 1]++;
    for (int e = 0; e < Mt; e++) for (int k = 0; k < 3; k++) m->inc_ptr[tris[3 * e + k] + 1]++;
    for (int e = 0; e < Mh; e++) for (int k = 0; k < 4; k++) m->inc_ptr[hinges[4 * e + k] + 1]++;
    for (int i = 0; i < N; i++) m->inc_ptr[i + 1] += m->inc_ptr[i];
    int *fill = (int *)calloc(N ? N : 1, sizeof(int));
    for (int e = 0; e < M; e++) for (int k = 0; k < 4; k++) { int i = tets[4 * e + k]; m->inc_slot[m->inc_ptr[i] + fill[i]++] = 4 * e + k; }
    for (int e = 0; e < Mt; e++) for (int k = 0; k < 3; k++) { int i = tris[3 * e + k]; m->inc_slot[m->inc_ptr[i] + fill[i]++] = 4 * M + 3 * e + k; }
    for (int e = 0; e < Mh; e++) for (int k = 0; k < 4; k++) { int i = hinges[4 * e + k]; m->inc_slot[m->inc_ptr[i] + fill[i]++] = 4 * M + 3 * Mt + 4 * e + k; }
    free(fill);
    return m;
}

/* read back rest-shape quantities (for pin tests) */
void orc_get_rest(const orc_model *m, double *tet_B, double *tet_V, double *tri_B, double *tri_A, double *theta0, double *l0) {
    if (tet_B) memcpy(tet_B, m->tet_B, sizeof(double) * 9 * m->M);
    if (tet_V) memcpy(tet_V, m->tet_V, sizeof(double) * m->M);
    if (tri_B) memcpy(tri_B, m->tri_B, sizeof(double) * 4 * m->Mt);
    if (tri_A) memcpy(tri_A, m->tri_A, sizeof(double) * m->Mt);
    if (theta0) memcpy(theta0, m->hinge_theta0, sizeof(double) * m->Mh);
    if (l0) memcpy(l0, m->hinge_l0, sizeof(double) * m->Mh);
}

/* set one parameter group for all envs; group: 0 tet_mu 1 tet_lambda 2 tet_damp 3 tri_mu 4 tri_lambda 5 tri_damp 6 mass
   7 hinge_kb (shared by all environments: row 0 of v is taken) */
int orc_set_params(orc_model *m, int group, const double *v) {
    double *dst[7] = {m->tet_mu, m->tet_lambda, m->tet_damp, m->tri_mu, m->tri_lambda, m->tri_damp, m->mass};
    size_t n[7] = {(size_t)m->M, (size_t)m->M, (size_t)m->M, (size_t)m->Mt, (size_t)m->Mt, (size_t)m->Mt, (size_t)m->N};
    if (group == 7) { memcpy(m->hinge_kb, v, sizeof(double) * m->Mh); return 0; }
    if (group >= 8 && group <= 11) { /* 8 ke 9 kd 10 kf 11 mu_c: one value per environment */
        double *cd[4] = {m->ke, m->kd, m->kf, m->mu_c};
        memcpy(cd[group - 8], v, sizeof(double) * m->E);
        return 0;
    }
    if (group == 12) { m->g[0] = v[0]; m->g[1] = v[1]; m->g[2] = v[2]; return 0; } /* gravity: one vector for all environments */
    if (group == 13) { memcpy(m->hinge_theta0, v, sizeof(double) * m->Mh); return 0; } /* rest angles: one array for all environments */
    if (group == 14) { memcpy(m->k_drag, v, sizeof(double) * m->E); return 0; }        /* one value per environment */
    if (group == 15) { memcpy(m->k_lift, v, sizeof(double) * m->E); return 0; }
    if (group == 16) { m->wind[0] = v[0]; m->wind[1] = v[1]; m->wind[2] = v[2]; return 0; } /* one vector for all environments; no gradient */
    if (group < 0 || group > 6) return -1;
    memcpy(dst[group], v, sizeof(double) * n[group] * m->E);
    return 0;
}
int orc_get_grads(const orc_model *m, int group, double *out) {
    const double *src[8] = {m->g_tet_mu, m->g_tet_lambda, m->g_tet_damp, m->g_tri_mu, m->g_tri_lambda, m->g_tri_damp, m->g_mass, m->g_hinge_kb};
    size_t n[8] = {(size_t)m->M, (size_t)m->M, (size_t)m->M, (size_t)m->Mt, (size_t)m->Mt, (size_t)m->Mt, (size_t)m->N, (size_t)m->Mh};
    if (group >= 8 && group <= 11) {
        const double *cs[4] = {m->g_ke, m->g_kd, m->g_kf, m->g_muc};
        memcpy(out, cs[group - 8], sizeof(double) * m->E);
        return 0;
    }
    if (group == 12) { memcpy(out, m->g_gravity, sizeof(double) * 3 * m->E); return 0; } /* [E][3] */
    if (group == 13) { memcpy(out, m->g_hinge_theta0, sizeof(double) * m->Mh * m->E); return 0; } /* [E][Mh] */
    if (group == 14) { memcpy(out, m->g_kdrag, sizeof(double) * m->E); return 0; }
    if (group == 15) { memcpy(out, m->g_klift, sizeof(double) * m->E); return 0; }
    if (group == 100) { memcpy(out, m->g_con_abs, sizeof(double) * 4 * m->E); return 0; } /* [E][4] diagnostic */
    if (group < 0 || group > 7) return -1;
    memcpy(out, src[group], sizeof(double) * n[group] * m->E);
    return 0;
}
void orc_zero_grads(orc_model *m) {
    size_t E = m->E;
    memset(m->g_tet_mu, 0, sizeof(double) * E * m->M); memset(m->g_tet_lambda, 0, sizeof(double) * E * m->M); memset(m->g_tet_damp, 0, sizeof(double) * E * m->M);
    memset(m->g_tri_mu, 0, sizeof(double) * E * m->Mt); memset(m->g_tri_lambda, 0, sizeof(double) * E * m->Mt); memset(m->g_tri_damp, 0, sizeof(double) * E * m->Mt);
    memset(m->g_mass, 0, sizeof(double) * E * m->N);
    memset(m->g_hinge_kb, 0, sizeof(double) * E * m->Mh);
    memset(m->g_ke, 0, sizeof(double) * E); memset(m->g_kd, 0, sizeof(double) * E); memset(m->g_kf, 0, sizeof(double) * E); memset(m->g_muc, 0, sizeof(double) * E);
    memset(m->g_gravity, 0, sizeof(double) * E * 3); memset(m->g_con_abs, 0, sizeof(double) * E * 4);
    memset(m->g_kdrag, 0, sizeof(double) * E); memset(m->g_klift, 0, sizeof(double) * E);
    memset(m->g_tet_act, 0, sizeof(double) * E * m->M); memset(m->g_hinge_act, 0, sizeof(double) * E * m->Mh);
    memset(m->g_hinge_theta0, 0, sizeof(double) * E * m->Mh);
    if (m->g_sched_tet) memset(m->g_sched_tet, 0, sizeof(double) * m->act_frames * E * m->M);
    if (m->g_sched_hinge) memset(m->g_sched_hinge, 0, sizeof(double) * m->act_frames * E * m->Mh);
}

/* ---------------------------------------------------------------- tets */
/* Psi = mu/2 (I_C - 3) + lambda/2 (J - alpha)^2 - mu/2 log(I_C + 1), alpha = 1 + 3mu/(4 lambda) (A1) */
static void tet_kin(const double *x[4], const double *B, double *F) {
    double Ds[9], c[3];
    for (int k = 0; k < 3; k++) { v_sub(x[k + 1], x[0], c); m_setcol(Ds, k, c); }
    m_mul(Ds, B, F);
}
static double tet_energy(const double *x[4], const double *B, double V, double mu, double lam, double act) {
    double F[9]; tet_kin(x, B, F);
    double Ic = m_ddot(F, F), J = m_det(F), alpha = 1.0 + 0.75 * mu / lam + act; /* A1: passive alpha + actuation */
    return V * (0.5 * mu * (Ic - 3.0) + 0.5 * lam * (J - alpha) * (J - alpha) - 0.5 * mu * log(Ic + 1.0));
}
/* first Piola-Kirchhoff stress P = dPsi/dF + damping stress k F sym(F^T Fdot) (A3); also returns the
   three parameter directions Pmu, Plam, Pk with P = mu Pmu + lam Plam + k Pk */
static void tet_stress(const double *F, const double *Fd, double mu, double lam, double kd, double act, double *P, double *Pmu, double *Plam, double *Pk) {
    double C[9], S[9], T[9], pm[9], pl[9], pk[9];
    double Ic = m_ddot(F, F), J = m_det(F);
    m_cof(F, C);
    double s1 = 1.0 - 1.0 / (Ic + 1.0);
    for (int i = 0; i < 9; i++) { pm[i] = s1 * F[i] - 0.75 * C[i]; pl[i] = (J - 1.0 - act) * C[i]; } /* lambda (J - alpha) cof F, alpha = 1 + 3mu/(4 lambda) + act */
    m_mul_tn(F, Fd, T); m_sym(T, S); m_mul(F, S, pk);
    for (int i = 0; i < 9; i++) P[i] = mu * pm[i] + lam * pl[i] + kd * pk[i];
    if (Pmu) memcpy(Pmu, pm, sizeof pm);
    if (Plam) memcpy(Plam, pl, sizeof pl);
    if (Pk) memcpy(Pk, pk, sizeof pk);
}
/* nodal forces: H = -V P B^T, f_{1..3} = columns of H, f_0 = -(sum) */
static void tet_force(const double *x[4], const double *v[4], const double *B, double V, double mu, double lam, double kd, double act, double f[4][3]) {
    double F[9], Fd[9], P[9], H[9];
    tet_kin(x, B, F); tet_kin(v, B, Fd);
    tet_stress(F, Fd, mu, lam, kd, act, P, NULL, NULL, NULL);
    m_mul_nt(P, B, H);
    f[0][0] = f[0][1] = f[0][2] = 0;
    for (int k = 0; k < 3; k++) {
        double c[3]; m_col(H, k, c);
        v_scale(-V, c, f[k + 1]);
        v_axpy(-1.0, f[k + 1], f[0]);
    }
}
/* VJP: given a_k = dL/df_k, add to ax_k = dL/dx_k, av_k = dL/dv_k, and parameter gradients */
static void tet_adjoint(const double *x[4], const double *v[4], const double *a[4], const double *B, double V, double mu, double lam, double kd, double act,
                        double ax[4][3], double av[4][3], double *gmu, double *glam, double *gk, double *gact) {
    double F[9], Fd[9], P[9], Pmu[9], Plam[9], Pk[9], G[9], A[9], c[3];
    tet_kin(x, B, F); tet_kin(v, B, Fd);
    tet_stress(F, Fd, mu, lam, kd, act, P, Pmu, Plam, Pk);
    for (int k = 0; k < 3; k++) { v_sub(a[k + 1], a[0], c); m_setcol(G, k, c); }
    m_mul(G, B, A);
    for (int i = 0; i < 9; i++) A[i] *= -V; /* A = adj_P = -V G B */
    *gmu += m_ddot(Pmu, A); *glam += m_ddot(Plam, A); *gk += m_ddot(Pk, A);
    /* adj_F = (dP/dF)^T[A]; the elastic Hessian is symmetric */
    double C[9], D[9], aF[9], aFd[9], S[9], Nn[9], T[9], T2[9];
    double Ic = m_ddot(F, F), J = m_det(F), alpha = 1.0 + 0.75 * mu / lam + act;
    m_cof(F, C); m_dcof(F, A, D);
    double s1 = 1.0 - 1.0 / (Ic + 1.0), FA = m_ddot(F, A), CA = m_ddot(C, A);
    *gact += -lam * CA; /* dP/d(act) = -lambda cof F */
    for (int i = 0; i < 9; i++)
        aF[i] = mu * s1 * A[i] + 2.0 * mu * FA / ((Ic + 1.0) * (Ic + 1.0)) * F[i] + lam * CA * C[i] + lam * (J - alpha) * D[i];
    /* damping P_d = k F S, S = sym(F^T Fd): adj_F += k (A S + Fd N), adj_Fd = k F N, N = sym(F^T A) */
    m_mul_tn(F, Fd, T); m_sym(T, S); m_mul_tn(F, A, T); m_sym(T, Nn);
    m_mul(A, S, T); m_mul(Fd, Nn, T2);
    for (int i = 0; i < 9; i++) aF[i] += kd * (T[i] + T2[i]);
    m_mul(F, Nn, aFd);
    for (int i = 0; i < 9; i++) aFd[i] *= kd;
    /* F = D_s B  =>  adj_Ds = adj_F B^T */
    double aDs[9], aDv[9];
    m_mul_nt(aF, B, aDs); m_mul_nt(aFd, B, aDv);
    for (int k = 0; k < 3; k++) {
        m_col(aDs, k, c); v_axpy(1.0, c, ax[k + 1]); v_axpy(-1.0, c, ax[0]);
        m_col(aDv, k, c); v_axpy(1.0, c, av[k + 1]); v_axpy(-1.0, c, av[0]);
    }
}

/* ---------------------------------------------------------------- triangles (A4) */
/* F (3x2) stored as two columns f1, f2 */
static void tri_kin(const double *x[3], const double *B, double f1[3], double f2[3]) {
    double e1[3], e2[3];
    v_sub(x[1], x[0], e1); v_sub(x[2], x[0], e2);
    for (int r = 0; r < 3; r++) { f1[r] = e1[r] * B[0] + e2[r] * B[2]; f2[r] = e1[r] * B[1] + e2[r] * B[3]; }
}
static double tri_energy(const double *x[3], const double *B, double A, double mu, double lam) {
    double f1[3], f2[3], c[3]; tri_kin(x, B, f1, f2);
    double Ic = v_dot(f1, f1) + v_dot(f2, f2);
    v_cross(f1, f2, c);
    double J = sqrt(v_dot(c, c)), alpha = 1.0 + 2.0 * mu / (3.0 * lam);
    return A * (0.5 * mu * (Ic - 2.0) + 0.5 * lam * (J - alpha) * (J - alpha) - 0.5 * mu * log(Ic + 1.0));
}
/* P (3x2) as columns p1, p2; parameter directions like the tet */
static void tri_stress(const double f1[3], const double f2[3], const double g1[3], const double g2[3], double mu, double lam, double kd,
                       double p1[3], double p2[3], double pm[2][3], double pl[2][3], double pk[2][3]) {
    double c[3], n[3], j1[3], j2[3];
    double Ic = v_dot(f1, f1) + v_dot(f2, f2);
    v_cross(f1, f2, c);
    double J = sqrt(v_dot(c, c));
    v_scale(1.0 / fmax(J, 1e-12), c, n);
    v_cross(f2, n, j1); v_cross(n, f1, j2); /* dJ/dF = [f2 x n, n x f1] */
    double s1 = 1.0 - 1.0 / (Ic + 1.0);
    /* S = sym(F^T Fdot) 2x2 */
    double s11 = v_dot(f1, g1), s22 = v_dot(f2, g2), s12 = 0.5 * (v_dot(f1, g2) + v_dot(f2, g1));
    for (int r = 0; r < 3; r++) {
        pm[0][r] = s1 * f1[r] - (2.0 / 3.0) * j1[r]; pm[1][r] = s1 * f2[r] - (2.0 / 3.0) * j2[r];
        pl[0][r] = (J - 1.0) * j1[r]; pl[1][r] = (J - 1.0) * j2[r];
        pk[0][r] = f1[r] * s11 + f2[r] * s12; pk[1][r] = f1[r] * s12 + f2[r] * s22;
        p1[r] = mu * pm[0][r] + lam * pl[0][r] + kd * pk[0][r];
        p2[r] = mu * pm[1][r] + lam * pl[1][r] + kd * pk[1][r];
    }
}
/* H = -A P B^T (3x2): h1 = -A (p1 B00 + p2 B01), h2 = -A (p1 B10 + p2 B11) */
static void tri_force(const double *x[3], const double *v[3], const double *B, double A, double mu, double lam, double kd, double f[3][3]) {
    double f1[3], f2[3], g1[3], g2[3], p1[3], p2[3], pm[2][3], pl[2][3], pk[2][3];
    tri_kin(x, B, f1, f2); tri_kin(v, B, g1, g2);
    tri_stress(f1, f2, g1, g2, mu, lam, kd, p1, p2, pm, pl, pk);
    for (int r = 0; r < 3; r++) {
        f[1][r] = -A * (p1[r] * B[0] + p2[r] * B[1]);
        f[2][r] = -A * (p1[r] * B[2] + p2[r] * B[3]);
        f[0][r] = -(f[1][r] + f[2][r]);
    }
}
static void tri_adjoint(const double *x[3], const double *v[3], const double *a[3], const double *B, double A, double mu, double lam, double kd,
                        double ax[3][3], double av[3][3], double *gmu, double *glam, double *gk) {
    double f1[3], f2[3], g1[3], g2[3], p1[3], p2[3], pm[2][3], pl[2][3], pk[2][3];
    tri_kin(x, B, f1, f2); tri_kin(v, B, g1, g2);
    tri_stress(f1, f2, g1, g2, mu, lam, kd, p1, p2, pm, pl, pk);
    /* A_ = adj_P = -A G B, G = [a1-a0, a2-a0] */
    double G1[3], G2[3], A1[3], A2[3];
    v_sub(a[1], a[0], G1); v_sub(a[2], a[0], G2);
    for (int r = 0; r < 3; r++) { A1[r] = -A * (G1[r] * B[0] + G2[r] * B[2]); A2[r] = -A * (G1[r] * B[1] + G2[r] * B[3]); }
    *gmu += v_dot(pm[0], A1) + v_dot(pm[1], A2);
    *glam += v_dot(pl[0], A1) + v_dot(pl[1], A2);
    *gk += v_dot(pk[0], A1) + v_dot(pk[1], A2);
    double c[3], n[3], j1[3], j2[3], dc[3], dn[3], t[3], t2[3];
    double Ic = v_dot(f1, f1) + v_dot(f2, f2);
    v_cross(f1, f2, c);
    double J = sqrt(v_dot(c, c)), Jg = fmax(J, 1e-12), alpha = 1.0 + 2.0 * mu / (3.0 * lam);
    v_scale(1.0 / Jg, c, n);
    v_cross(f2, n, j1); v_cross(n, f1, j2);
    double s1 = 1.0 - 1.0 / (Ic + 1.0);
    double FA = v_dot(f1, A1) + v_dot(f2, A2), JA = v_dot(j1, A1) + v_dot(j2, A2);
    /* D(dJ/dF)[A_] = [a2 x n + f2 x dn, dn x f1 + n x a1], dc = a1 x f2 + f1 x a2, dn = (dc - n (n.dc))/J */
    v_cross(A1, f2, dc); v_cross(f1, A2, t); dc[0] += t[0]; dc[1] += t[1]; dc[2] += t[2];
    double ndc = v_dot(n, dc);
    for (int r = 0; r < 3; r++) dn[r] = (dc[r] - n[r] * ndc) / Jg;
    double D1[3], D2[3];
    v_cross(A2, n, D1); v_cross(f2, dn, t); D1[0] += t[0]; D1[1] += t[1]; D1[2] += t[2];
    v_cross(dn, f1, D2); v_cross(n, A1, t2); D2[0] += t2[0]; D2[1] += t2[1]; D2[2] += t2[2];
    double aF1[3], aF2[3], aG1[3], aG2[3];
    double q = 2.0 * mu * FA / ((Ic + 1.0) * (Ic + 1.0));
    for (int r = 0; r < 3; r++) {
        aF1[r] = mu * s1 * A1[r] + q * f1[r] + lam * JA * j1[r] + lam * (J - alpha) * D1[r];
        aF2[r] = mu * s1 * A2[r] + q * f2[r] + lam * JA * j2[r] + lam * (J - alpha) * D2[r];
    }
    /* damping: S = sym(F^T Fd), N = sym(F^T A_) (2x2) */
    double s11 = v_dot(f1, g1), s22 = v_dot(f2, g2), s12 = 0.5 * (v_dot(f1, g2) + v_dot(f2, g1));
    double n11 = v_dot(f1, A1), n22 = v_dot(f2, A2), n12 = 0.5 * (v_dot(f1, A2) + v_dot(f2, A1));
    for (int r = 0; r < 3; r++) {
        aF1[r] += kd * (A1[r] * s11 + A2[r] * s12 + g1[r] * n11 + g2[r] * n12);
        aF2[r] += kd * (A1[r] * s12 + A2[r] * s22 + g1[r] * n12 + g2[r] * n22);
        aG1[r] = kd * (f1[r] * n11 + f2[r] * n12);
        aG2[r] = kd * (f1[r] * n12 + f2[r] * n22);
    }
    /* F = D_s B => adj_Ds = adj_F B^T: col1 = aF1 B00 + aF2 B01, col2 = aF1 B10 + aF2 B11 */
    for (int r = 0; r < 3; r++) {
        double d1 = aF1[r] * B[0] + aF2[r] * B[1], d2 = aF1[r] * B[2] + aF2[r] * B[3];
        ax[1][r] += d1; ax[2][r] += d2; ax[0][r] -= d1 + d2;
        double w1 = aG1[r] * B[0] + aG2[r] * B[1], w2 = aG1[r] * B[2] + aG2[r] * B[3];
        av[1][r] += w1; av[2][r] += w2; av[0][r] -= w1 + w2;
    }
}

/* ---------------------------------------------------------------- lift / drag on triangles (reading A21) */
/* Thin-plate model, quadratic in the speed: with c = (x1-x0) x (x2-x0), area A = |c|/2, unit normal n = c/|c|, relative
   velocity vb = (v0+v1+v2)/3 - wind, s = sqrt(|vb|^2 + eps^2) (eps = 1e-6 m/s keeps the model smooth at rest), v_n = n.vb:
       F = -A s (k_drag vb + k_lift v_n n)
   an isotropic drag plus a pressure term along the face normal (the part of it perpendicular to the flow is the lift of an
   inclined face); F is shared equally by the three vertices.  Dissipative: F.vb = -A s (k_drag |vb|^2 + k_lift v_n^2) <= 0. */
#define ORC_AERO_EPS 1e-6
static void aero_force(const double *x[3], const double *v[3], const double *wind, double kdrag, double klift, double f[3][3]) {
    double e1[3], e2[3], c[3], vb[3];
    v_sub(x[1], x[0], e1); v_sub(x[2], x[0], e2); v_cross(e1, e2, c);
    double L = sqrt(v_dot(c, c));
    for (int r = 0; r < 3; r++) vb[r] = (v[0][r] + v[1][r] + v[2][r]) / 3.0 - wind[r];
    double s = sqrt(v_dot(vb, vb) + ORC_AERO_EPS * ORC_AERO_EPS), A = 0.5 * L, vn = v_dot(c, vb) / L;
    for (int r = 0; r < 3; r++) {
        double F = -A * s * (kdrag * vb[r] + klift * vn * c[r] / L);
        f[0][r] = f[1][r] = f[2][r] = F / 3.0;
    }
}
/* VJP: a_k = dL/df_k.  Adds to ax, av and to the parameter gradients.  With ab = (a0+a1+a2)/3, L = |c|, u = c.vb,
   P = k_drag L vb + k_lift u c / L (F = -s P / 2):
     dL/dvb = -(ab.P)/(2 s) vb - (s/2) k_drag L ab - (s/2) k_lift (ab.c)/L c                       (shared: each dL/dv_k gets a third)
     dL/dc  = -(s/2) k_drag (ab.vb) n - (s/2) k_lift [ (ab.c)/L vb + (u/L) ab - u (ab.c)/L^2 n ]
     dL/de1 = e2 x dL/dc, dL/de2 = dL/dc x e1 */
static void aero_adjoint(const double *x[3], const double *v[3], const double *a[3], const double *wind, double kdrag, double klift,
                         double ax[3][3], double av[3][3], double *g_kdrag, double *g_klift) {
    double e1[3], e2[3], c[3], vb[3], ab[3], n[3], P[3], gv[3], gc[3], t1[3], t2[3];
    v_sub(x[1], x[0], e1); v_sub(x[2], x[0], e2); v_cross(e1, e2, c);
    double L = sqrt(v_dot(c, c));
    for (int r = 0; r < 3; r++) { vb[r] = (v[0][r] + v[1][r] + v[2][r]) / 3.0 - wind[r]; ab[r] = (a[0][r] + a[1][r] + a[2][r]) / 3.0; n[r] = c[r] / L; }
    double s = sqrt(v_dot(vb, vb) + ORC_AERO_EPS * ORC_AERO_EPS), u = v_dot(c, vb), ac = v_dot(ab, c), avb = v_dot(ab, vb);
    for (int r = 0; r < 3; r++) P[r] = kdrag * L * vb[r] + klift * u * c[r] / L;
    double aP = v_dot(ab, P);
    *g_kdrag += -0.5 * s * L * avb;
    *g_klift += -0.5 * s * u * ac / L;
    for (int r = 0; r < 3; r++) {
        gv[r] = -0.5 * aP / s * vb[r] - 0.5 * s * kdrag * L * ab[r] - 0.5 * s * klift * ac / L * c[r];
        gc[r] = -0.5 * s * kdrag * avb * n[r] - 0.5 * s * klift * (ac / L * vb[r] + u / L * ab[r] - u * ac / (L * L) * n[r]);
    }
    v_cross(e2, gc, t1); v_cross(gc, e1, t2);
    for (int r = 0; r < 3; r++) {
        ax[1][r] += t1[r]; ax[2][r] += t2[r]; ax[0][r] -= t1[r] + t2[r];
        av[0][r] += gv[r] / 3.0; av[1][r] += gv[r] / 3.0; av[2][r] += gv[r] / 3.0;
    }
}

/* ---------------------------------------------------------------- hinges (A5, A6) */
/* E_b = 2 k_b l0 (1 - cos((theta - theta0)/2)),  f_i = k_b l0 sin((theta - theta0)/2) d_i */
static double hinge_energy(const double *x[4], double theta0, double l0, double kb, double act) {
    double th = hinge_angle(x[0], x[1], x[2], x[3], NULL);
    return 2.0 * kb * l0 * (1.0 - cos(0.5 * (th - theta0) + act));
}
/* f_i = k_b l0 sin(phi/2 + alpha) d_i, phi = theta - theta0, alpha = the per-edge actuation */
static void hinge_force(const double *x[4], double theta0, double l0, double kb, double act, double f[4][3]) {
    double d[4][3];
    double th = hinge_angle(x[0], x[1], x[2], x[3], d);
    double s = kb * l0 * sin(0.5 * (th - theta0) + act);
    for (int k = 0; k < 4; k++) v_scale(s, d[k], f[k]);
}
/* VJP = JVP (conservative force, symmetric Jacobian): adj_x_j += -E'' s d_j + E' Dd_j[a], s = sum d_i.a_i */
/* f_i = k_b l0 sin(ph) d_i is linear in k_b: dL/dk_b += l0 sin(ph) sum_i d_i . a_i */
/* dL/d(alpha) += k_b l0 cos(ph) sum_i d_i . a_i; the rest angle enters as -theta0/2 in the same argument: dL/d(theta0) = -1/2 of that */
static void hinge_adjoint(const double *x[4], const double *a[4], double theta0, double l0, double kb, double act, double ax[4][3], double *g_kb,
                          double *g_act, double *g_theta0) {
    const double *x1 = x[0], *x2 = x[1], *x3 = x[2], *x4 = x[3];
    double p13[3], p14[3], p23[3], p24[3], n1[3], n2[3], e[3], eh[3];
    v_sub(x1, x3, p13); v_sub(x1, x4, p14); v_sub(x2, x3, p23); v_sub(x2, x4, p24);
    v_cross(p13, p14, n1); v_cross(p24, p23, n2); v_sub(x4, x3, e);
    double L = sqrt(v_dot(e, e)), n1s = v_dot(n1, n1), n2s = v_dot(n2, n2);
    v_scale(1.0 / L, e, eh);
    double m1[3], m2[3], d[4][3];
    v_scale(1.0 / n1s, n1, m1); v_scale(1.0 / n2s, n2, m2);
    double c13 = v_dot(p13, eh), c14 = v_dot(p14, eh), c23 = v_dot(p23, eh), c24 = v_dot(p24, eh);
    double th = hinge_angle(x1, x2, x3, x4, d);
    /* tangents along a */
    double q13[3], q14[3], q23[3], q24[3], dn1[3], dn2[3], de[3], deh[3], t[3];
    v_sub(a[0], a[2], q13); v_sub(a[0], a[3], q14); v_sub(a[1], a[2], q23); v_sub(a[1], a[3], q24);
    v_cross(q13, p14, dn1); v_cross(p13, q14, t); dn1[0] += t[0]; dn1[1] += t[1]; dn1[2] += t[2];
    v_cross(q24, p23, dn2); v_cross(p24, q23, t); dn2[0] += t[0]; dn2[1] += t[1]; dn2[2] += t[2];
    v_sub(a[3], a[2], de);
    double dL = v_dot(eh, de);
    for (int r = 0; r < 3; r++) deh[r] = (de[r] - eh[r] * dL) / L;
    double dm1[3], dm2[3];
    double k1 = v_dot(n1, dn1), k2 = v_dot(n2, dn2);
    for (int r = 0; r < 3; r++) {
        dm1[r] = dn1[r] / n1s - 2.0 * n1[r] * k1 / (n1s * n1s);
        dm2[r] = dn2[r] / n2s - 2.0 * n2[r] * k2 / (n2s * n2s);
    }
    double dc13 = v_dot(q13, eh) + v_dot(p13, deh), dc14 = v_dot(q14, eh) + v_dot(p14, deh);
    double dc23 = v_dot(q23, eh) + v_dot(p23, deh), dc24 = v_dot(q24, eh) + v_dot(p24, deh);
    double dd[4][3];
    for (int r = 0; r < 3; r++) {
        dd[0][r] = dL * m1[r] + L * dm1[r];
        dd[1][r] = dL * m2[r] + L * dm2[r];
        dd[2][r] = dc14 * m1[r] + c14 * dm1[r] + dc24 * m2[r] + c24 * dm2[r];
        dd[3][r] = -(dc13 * m1[r] + c13 * dm1[r] + dc23 * m2[r] + c23 * dm2[r]);
    }
    double s = 0;
    for (int k = 0; k < 4; k++) s += v_dot(d[k], a[k]);
    double ph = 0.5 * (th - theta0) + act;
    double E1 = kb * l0 * sin(ph), E2 = 0.5 * kb * l0 * cos(ph);
    for (int k = 0; k < 4; k++) for (int r = 0; r < 3; r++) ax[k][r] += -E2 * s * d[k][r] + E1 * dd[k][r];
    if (g_kb) *g_kb += l0 * sin(ph) * s;
    if (g_act) *g_act += 2.0 * E2 * s;
    if (g_theta0) *g_theta0 += -E2 * s;
}

/* ---------------------------------------------------------------- contact (A7, A8) */
static void contact_force(const orc_model *m, int env, const double *x, const double *v, double f[3]) {
    f[0] = f[1] = f[2] = 0;
    double c = v_dot(m->n, x) - m->d - m->r;
    if (!(c < 0)) return;
    double vn = v_dot(m->n, v);
    double fn = -m->ke[env] * c - m->kd[env] * fmin(vn, 0.0);
    double vt[3] = {v[0] - m->n[0] * vn, v[1] - m->n[1] * vn, v[2] - m->n[2] * vn};
    double s = sqrt(v_dot(vt, vt));
    double coef = fmin(m->kf[env], m->mu_c[env] * fn / fmax(s, 1e-12));
    for (int r = 0; r < 3; r++) f[r] = m->n[r] * fn - coef * vt[r];
}
/* gp[4] (may be NULL): this particle's contributions to dL/dk_e, dL/dk_d, dL/dk_f, dL/dmu_c.  With a.f = f_n afn (afn as
   below): d/dk_e = -c afn, d/dk_d = -min(v_n, 0) afn; stick: d/dk_f = -(v_t.a_t); slip: d/dmu_c = -f_n (v_t.a_t)/s */
static void contact_adjoint(const orc_model *m, int env, const double *x, const double *v, const double *a, double ax[3], double av[3], double *gp) {
    if (gp) gp[0] = gp[1] = gp[2] = gp[3] = 0.0;
    double c = v_dot(m->n, x) - m->d - m->r;
    if (!(c < 0)) return;
    const double *n = m->n;
    double vn = v_dot(n, v);
    double fn = -m->ke[env] * c - m->kd[env] * fmin(vn, 0.0);
    double vt[3] = {v[0] - n[0] * vn, v[1] - n[1] * vn, v[2] - n[2] * vn};
    double s = sqrt(v_dot(vt, vt)), sg = fmax(s, 1e-12);
    double na = v_dot(n, a);
    double at[3] = {a[0] - n[0] * na, a[1] - n[1] * na, a[2] - n[2] * na};
    double afn, avt[3];
    double kf = m->kf[env], muc = m->mu_c[env];
    if (muc * fn / sg >= kf) { /* stick: f_f = -k_f v_t */
        afn = na;
        v_scale(-kf, at, avt);
        if (gp) gp[2] = -v_dot(vt, at);
    } else { /* slip: f_f = -mu_c f_n v_t / s */
        double vta = v_dot(vt, at);
        afn = na - muc * vta / sg;
        if (gp) gp[3] = -fn * vta / sg;
        for (int r = 0; r < 3; r++) avt[r] = -muc * fn * (at[r] / sg - vt[r] * vta / (sg * sg * sg));
    }
    if (gp) { gp[0] = -c * afn; gp[1] = -fmin(vn, 0.0) * afn; }
    v_axpy(1.0, avt, av);
    v_axpy(-m->ke[env] * afn, n, ax);
    if (vn < 0) v_axpy(-m->kd[env] * afn, n, av);
}

/* ---------------------------------------------------------------- forces on one environment */
enum { ORC_TETS = 1, ORC_TRIS = 2, ORC_HINGES = 4, ORC_CONTACT = 8, ORC_ALL = 15 };

/* f[N][3] = sum of the selected force terms at state (x, v) of environment env; slots is scratch [n_slots][3] */
static void env_forces(const orc_model *m, int env, const double *x, const double *v, double *f, double *slots, int mask, int par) {
    const int N = m->N, M = m->M, Mt = m->Mt, Mh = m->Mh;
    memset(slots, 0, sizeof(double) * 3 * (m->n_slots ? m->n_slots : 1));
    if (mask & ORC_TETS) {
#pragma omp parallel for if (par) schedule(static)
        for (int e = 0; e < M; e++) {
            const int *t = m->tets + 4 * e;
            const double *xe[4], *ve[4];
            for (int k = 0; k < 4; k++) { xe[k] = x + 3 * t[k]; ve[k] = v + 3 * t[k]; }
            double fe[4][3];
            tet_force(xe, ve, m->tet_B + 9 * e, m->tet_V[e], m->tet_mu[(size_t)env * M + e], m->tet_lambda[(size_t)env * M + e], m->tet_damp[(size_t)env * M + e], m->tet_act[(size_t)env * M + e], fe);
            memcpy(slots + 3 * (4 * (size_t)e), fe, sizeof fe);
        }
    }
    if (mask & ORC_TRIS) {
#pragma omp parallel for if (par) schedule(static)
        for (int e = 0; e < Mt; e++) {
            const int *t = m->tris + 3 * e;
            const double *xe[3], *ve[3];
            for (int k = 0; k < 3; k++) { xe[k] = x + 3 * t[k]; ve[k] = v + 3 * t[k]; }
            double fe[3][3];
            tri_force(xe, ve, m->tri_B + 4 * e, m->tri_A[e], m->tri_mu[(size_t)env * Mt + e], m->tri_lambda[(size_t)env * Mt + e], m->tri_damp[(size_t)env * Mt + e], fe);
            if (m->k_drag[env] != 0.0 || m->k_lift[env] != 0.0) { /* lift / drag of the air on this face */
                double fa[3][3];
                aero_force(xe, ve, m->wind, m->k_drag[env], m->k_lift[env], fa);
                for (int k = 0; k < 3; k++) v_axpy(1.0, fa[k], fe[k]);
            }
            memcpy(slots + 3 * (4 * (size_t)M + 3 * (size_t)e), fe, sizeof fe);
        }
    }
    if (mask & ORC_HINGES) {
#pragma omp parallel for if (par) schedule(static)
        for (int e = 0; e < Mh; e++) {
            const int *h = m->hinges + 4 * e;
            const double *xe[4];
            for (int k = 0; k < 4; k++) xe[k] = x + 3 * h[k];
            double fe[4][3];
            hinge_force(xe, m->hinge_theta0[e], m->hinge_l0[e], m->hinge_kb[e], m->hinge_act[(size_t)env * Mh + e], fe);
            memcpy(slots + 3 * (4 * (size_t)M + 3 * (size_t)Mt + 4 * (size_t)e), fe, sizeof fe);
        }
    }
#pragma omp parallel for if (par) schedule(static)
    for (int i = 0; i < N; i++) {
        double fi[3] = {0, 0, 0};
        for (int q = m->inc_ptr[i]; q < m->inc_ptr[i + 1]; q++) v_axpy(1.0, slots + 3 * (size_t)m->inc_slot[q], fi);
        if (mask & ORC_CONTACT) {
            double fc[3];
            contact_force(m, env, x + 3 * i, v + 3 * i, fc);
            v_axpy(1.0, fc, fi);
        }
        f[3 * i] = fi[0]; f[3 * i + 1] = fi[1]; f[3 * i + 2] = fi[2];
    }
}

/* OpenMP inside one environment only pays for big meshes */
static int par_inside(const orc_model *m) { return m->n_slots + m->N > 20000; }

/* public: forces of selected terms for all envs: x, v, f are [E][N][3] */
void orc_forces(const orc_model *m, const double *x, const double *v, double *f, int mask) {
    double *slots = zeros_d(3 * (size_t)m->n_slots);
    for (int env = 0; env < m->E; env++) {
        size_t o = (size_t)env * m->N * 3;
        env_forces(m, env, x + o, v + o, f + o, slots, mask, par_inside(m));
    }
    free(slots);
}
/* public: elastic potential energy per env of the selected element types (no damping: not a potential) */
void orc_energy(const orc_model *m, const double *x, int mask, double *U) {
    for (int env = 0; env < m->E; env++) {
        const double *xe_ = x + (size_t)env * m->N * 3;
        double u = 0;
        if (mask & ORC_TETS) for (int e = 0; e < m->M; e++) {
            const int *t = m->tets + 4 * e; const double *xe[4];
            for (int k = 0; k < 4; k++) xe[k] = xe_ + 3 * t[k];
            u += tet_energy(xe, m->tet_B + 9 * e, m->tet_V[e], m->tet_mu[(size_t)env * m->M + e], m->tet_lambda[(size_t)env * m->M + e], m->tet_act[(size_t)env * m->M + e]);
        }
        if (mask & ORC_TRIS) for (int e = 0; e < m->Mt; e++) {
            const int *t = m->tris + 3 * e; const double *xe[3];
            for (int k = 0; k < 3; k++) xe[k] = xe_ + 3 * t[k];
            u += tri_energy(xe, m->tri_B + 4 * e, m->tri_A[e], m->tri_mu[(size_t)env * m->Mt + e], m->tri_lambda[(size_t)env * m->Mt + e]);
        }
        if (mask & ORC_HINGES) for (int e = 0; e < m->Mh; e++) {
            const int *h = m->hinges + 4 * e; const double *xe[4];
            for (int k = 0; k < 4; k++) xe[k] = xe_ + 3 * h[k];
            u += hinge_energy(xe, m->hinge_theta0[e], m->hinge_l0[e], m->hinge_kb[e], m->hinge_act[(size_t)env * m->Mh + e]);
        }
        U[env] = u;
    }
}

/* ---------------------------------------------------------------- substep */
static double inv_mass(const orc_model *m, int env, int i) { return m->pinned[i] ? 0.0 : 1.0 / m->mass[(size_t)env * m->N + i]; }

static void env_step(const orc_model *m, int env, const double *x, const double *v, double *xo, double *vo, double *f, double *slots, int par) {
    env_forces(m, env, x, v, f, slots, ORC_ALL, par);
#pragma omp parallel for if (par) schedule(static)
    for (int i = 0; i < m->N; i++) {
        double w = inv_mass(m, env, i), on = w > 0 ? 1.0 : 0.0;
        for (int r = 0; r < 3; r++) {
            double v1 = v[3 * i + r] + (f[3 * i + r] * w + m->g[r] * on) * m->dt; /* Listing 1 (sign of g: A10) */
            vo[3 * i + r] = v1;
            xo[3 * i + r] = x[3 * i + r] + v1 * m->dt;
        }
    }
}

void orc_step(const orc_model *m, const double *x, const double *v, double *xo, double *vo) {
    const size_t S = (size_t)m->N * 3;
    const int par_env = m->E > 1;
#pragma omp parallel for if (par_env) schedule(dynamic, 1)
    for (int env = 0; env < m->E; env++) {
        double *f = zeros_d(S), *slots = zeros_d(3 * (size_t)m->n_slots);
        env_step(m, env, x + env * S, v + env * S, xo + env * S, vo + env * S, f, slots, !par_env && par_inside(m));
        free(f); free(slots);
    }
}

/* adjoint of one substep of one env.  In: state (x,v) BEFORE the step, cotangents (bx,bv) of the state
   AFTER.  Out: cotangents (ax,av) of the state before.  Parameter gradients accumulate in the model. */
static void env_step_adjoint(orc_model *m, int env, const double *x, const double *v, const double *bx, const double *bv,
                             double *ax, double *av, double *f, double *af, double *slots, double *slots_v, int par) {
    const int N = m->N, M = m->M, Mt = m->Mt, Mh = m->Mh;
    const double dt = m->dt;
    env_forces(m, env, x, v, f, slots, ORC_ALL, par); /* total force of the forward step */
    double *gp = (double *)malloc(sizeof(double) * 4 * (size_t)(N ? N : 1)); /* per-particle contact-parameter contributions */
    /* 1. integrate: v+ = v + (f w + g [w>0]) dt, x+ = x + v+ dt */
#pragma omp parallel for if (par) schedule(static)
    for (int i = 0; i < N; i++) {
        double w = inv_mass(m, env, i);
        double lv[3], aw = 0;
        for (int r = 0; r < 3; r++) {
            lv[r] = bv[3 * i + r] + dt * bx[3 * i + r]; /* total cotangent of v+ */
            ax[3 * i + r] = bx[3 * i + r];
            av[3 * i + r] = lv[r];
            af[3 * i + r] = dt * w * lv[r];
            aw += dt * f[3 * i + r] * lv[r];
        }
        if (w > 0) m->g_mass[(size_t)env * N + i] += -w * w * aw; /* w = 1/m (A11) */
        /* 2. contact */
        contact_adjoint(m, env, x + 3 * i, v + 3 * i, af + 3 * i, ax + 3 * i, av + 3 * i, gp + 4 * (size_t)i);
    }
    /* gravity enters Listing 1 as v+ = v + (f w + g [w>0]) dt, so dL/dg = sum_i [w_i>0] dt lv_i (lv = cotangent of v+, = av here) */
    for (int i = 0; i < N; i++)
        if (inv_mass(m, env, i) > 0)
            for (int r = 0; r < 3; r++) m->g_gravity[(size_t)env * 3 + r] += dt * (bv[3 * i + r] + dt * bx[3 * i + r]);
    for (int i = 0; i < N; i++) { /* serial, particle order: independent of the thread count */
        m->g_ke[env] += gp[4 * (size_t)i]; m->g_kd[env] += gp[4 * (size_t)i + 1]; m->g_kf[env] += gp[4 * (size_t)i + 2]; m->g_muc[env] += gp[4 * (size_t)i + 3];
        for (int q = 0; q < 4; q++) m->g_con_abs[(size_t)env * 4 + q] += fabs(gp[4 * (size_t)i + q]);
    }
    free(gp);
    /* 3-5. elements: per-element-vertex contributions into private slots, then gather per particle */
    memset(slots, 0, sizeof(double) * 3 * (m->n_slots ? m->n_slots : 1));
    memset(slots_v, 0, sizeof(double) * 3 * (m->n_slots ? m->n_slots : 1));
#pragma omp parallel for if (par) schedule(static)
    for (int e = 0; e < M; e++) {
        const int *t = m->tets + 4 * e;
        const double *xe[4], *ve[4], *ae[4];
        for (int k = 0; k < 4; k++) { xe[k] = x + 3 * t[k]; ve[k] = v + 3 * t[k]; ae[k] = af + 3 * t[k]; }
        double cx[4][3] = {{0}}, cv[4][3] = {{0}};
        size_t pe = (size_t)env * M + e;
        tet_adjoint(xe, ve, ae, m->tet_B + 9 * e, m->tet_V[e], m->tet_mu[pe], m->tet_lambda[pe], m->tet_damp[pe], m->tet_act[pe], cx, cv,
                    &m->g_tet_mu[pe], &m->g_tet_lambda[pe], &m->g_tet_damp[pe], &m->g_tet_act[pe]);
        memcpy(slots + 3 * (4 * (size_t)e), cx, sizeof cx);
        memcpy(slots_v + 3 * (4 * (size_t)e), cv, sizeof cv);
    }
    const int aero = m->k_drag[env] != 0.0 || m->k_lift[env] != 0.0;
    double *gaero = aero ? zeros_d(2 * (size_t)Mt) : NULL; /* per-triangle terms of dL/dk_drag, dL/dk_lift, summed in element order below */
#pragma omp parallel for if (par) schedule(static)
    for (int e = 0; e < Mt; e++) {
        const int *t = m->tris + 3 * e;
        const double *xe[3], *ve[3], *ae[3];
        for (int k = 0; k < 3; k++) { xe[k] = x + 3 * t[k]; ve[k] = v + 3 * t[k]; ae[k] = af + 3 * t[k]; }
        double cx[3][3] = {{0}}, cv[3][3] = {{0}};
        size_t pe = (size_t)env * Mt + e;
        tri_adjoint(xe, ve, ae, m->tri_B + 4 * e, m->tri_A[e], m->tri_mu[pe], m->tri_lambda[pe], m->tri_damp[pe], cx, cv,
                    &m->g_tri_mu[pe], &m->g_tri_lambda[pe], &m->g_tri_damp[pe]);
        if (aero) aero_adjoint(xe, ve, ae, m->wind, m->k_drag[env], m->k_lift[env], cx, cv, &gaero[2 * (size_t)e], &gaero[2 * (size_t)e + 1]);
        memcpy(slots + 3 * (4 * (size_t)M + 3 * (size_t)e), cx, sizeof cx);
        memcpy(slots_v + 3 * (4 * (size_t)M + 3 * (size_t)e), cv, sizeof cv);
    }
    if (aero) {
        for (int e = 0; e < Mt; e++) { m->g_kdrag[env] += gaero[2 * (size_t)e]; m->g_klift[env] += gaero[2 * (size_t)e + 1]; }
        free(gaero);
    }
#pragma omp parallel for if (par) schedule(static)
    for (int e = 0; e < Mh; e++) {
        const int *h = m->hinges + 4 * e;
        const double *xe[4], *ae[4];
        for (int k = 0; k < 4; k++) { xe[k] = x + 3 * h[k]; ae[k] = af + 3 * h[k]; }
        double cx[4][3] = {{0}};
        size_t pe = (size_t)env * Mh + e;
        hinge_adjoint(xe, ae, m->hinge_theta0[e], m->hinge_l0[e], m->hinge_kb[e], m->hinge_act[pe], cx, &m->g_hinge_kb[pe], &m->g_hinge_act[pe], &m->g_hinge_theta0[pe]);
        memcpy(slots + 3 * (4 * (size_t)M + 3 * (size_t)Mt + 4 * (size_t)e), cx, sizeof cx);
    }
#pragma omp parallel for if (par) schedule(static)
    for (int i = 0; i < N; i++)
        for (int q = m->inc_ptr[i]; q < m->inc_ptr[i + 1]; q++) {
            v_axpy(1.0, slots + 3 * (size_t)m->inc_slot[q], ax + 3 * i);
            v_axpy(1.0, slots_v + 3 * (size_t)m->inc_slot[q], av + 3 * i);
        }
}

void orc_step_adjoint(orc_model *m, const double *x, const double *v, const double *bx, const double *bv, double *ax, double *av) {
    const size_t S = (size_t)m->N * 3;
    const int par_env = m->E > 1;
#pragma omp parallel for if (par_env) schedule(dynamic, 1)
    for (int env = 0; env < m->E; env++) {
        double *f = zeros_d(S), *af = zeros_d(S), *s1 = zeros_d(3 * (size_t)m->n_slots), *s2 = zeros_d(3 * (size_t)m->n_slots);
        env_step_adjoint(m, env, x + env * S, v + env * S, bx + env * S, bv + env * S, ax + env * S, av + env * S, f, af, s1, s2, !par_env && par_inside(m));
        free(f); free(af); free(s1); free(s2);
    }
}

/* ---------------------------------------------------------------- actuation inputs */
/* CURRENT activation of every tet / hinge, [E][M] / [E][Mh]; NULL leaves that kind as it is.  Used by orc_step,
   orc_step_adjoint, orc_forces, orc_energy. */
void orc_set_act_current(orc_model *m, const double *tet_act, const double *hinge_act) {
    if (tet_act) memcpy(m->tet_act, tet_act, sizeof(double) * m->E * m->M);
    if (hinge_act) memcpy(m->hinge_act, hinge_act, sizeof(double) * m->E * m->Mh);
}
/* dL/d(current activation) accumulated by the adjoint substeps since the last orc_zero_grads */
void orc_get_act_grads_current(const orc_model *m, double *g_tet, double *g_hinge) {
    if (g_tet) memcpy(g_tet, m->g_tet_act, sizeof(double) * m->E * m->M);
    if (g_hinge) memcpy(g_hinge, m->g_hinge_act, sizeof(double) * m->E * m->Mh);
}
/* Activation SCHEDULE of rollouts: n_frames frames, frame f holds during substeps [f stride, (f+1) stride) (the last
   frame holds to the end).  tet [F][E][M], hinge [F][E][Mh], either may be NULL; n_frames = 0 removes the schedule. */
void orc_set_act_schedule(orc_model *m, int n_frames, int stride, const double *tet, const double *hinge) {
    free(m->sched_tet); free(m->sched_hinge); free(m->g_sched_tet); free(m->g_sched_hinge);
    m->sched_tet = m->sched_hinge = m->g_sched_tet = m->g_sched_hinge = NULL;
    m->act_frames = n_frames; m->act_stride = stride > 0 ? stride : 1;
    if (n_frames <= 0) { m->act_frames = 0; return; }
    if (tet) { m->sched_tet = dup_d(tet, (size_t)n_frames * m->E * m->M); m->g_sched_tet = zeros_d((size_t)n_frames * m->E * m->M); }
    if (hinge) { m->sched_hinge = dup_d(hinge, (size_t)n_frames * m->E * m->Mh); m->g_sched_hinge = zeros_d((size_t)n_frames * m->E * m->Mh); }
}
void orc_get_act_schedule_grads(const orc_model *m, double *g_tet, double *g_hinge) {
    if (g_tet && m->g_sched_tet) memcpy(g_tet, m->g_sched_tet, sizeof(double) * m->act_frames * m->E * m->M);
    if (g_hinge && m->g_sched_hinge) memcpy(g_hinge, m->g_sched_hinge, sizeof(double) * m->act_frames * m->E * m->Mh);
}
static int act_frame_of(const orc_model *m, int t) { int f = t / m->act_stride; return f < m->act_frames ? f : m->act_frames - 1; }
/* the activation of substep t becomes current */
static void act_load(orc_model *m, int t) {
    if (m->act_frames <= 0) return;
    int f = act_frame_of(m, t);
    if (m->sched_tet) memcpy(m->tet_act, m->sched_tet + (size_t)f * m->E * m->M, sizeof(double) * m->E * m->M);
    if (m->sched_hinge) memcpy(m->hinge_act, m->sched_hinge + (size_t)f * m->E * m->Mh, sizeof(double) * m->E * m->Mh);
}
/* the gradient the adjoint of substep t just added to the current accumulators moves to the schedule's frame */
static void act_collect(orc_model *m, int t) {
    if (m->act_frames <= 0) return;
    int f = act_frame_of(m, t);
    size_t nt = (size_t)m->E * m->M, nh = (size_t)m->E * m->Mh;
    if (m->g_sched_tet) for (size_t i = 0; i < nt; i++) { m->g_sched_tet[f * nt + i] += m->g_tet_act[i]; m->g_tet_act[i] = 0; }
    if (m->g_sched_hinge) for (size_t i = 0; i < nh; i++) { m->g_sched_hinge[f * nh + i] += m->g_hinge_act[i]; m->g_hinge_act[i] = 0; }
}

/* ---------------------------------------------------------------- rollout + tape */
/* Forward T substeps from (x0, v0) [E][N][3].  Checkpoints: state after t substeps for t = 0, K, 2K, ... < T
   go to ck_x, ck_v [n_ck][E][N][3], n_ck = ceil(T/K)  (K = 1: the full tape).  States after rec_t[j]
   substeps (sorted ascending, 0 <= rec_t <= T) are copied to rec_x, rec_v [n_rec][E][N][3] (either may
   be NULL).  Final state to xT, vT (may be NULL). */
void orc_rollout(orc_model *m, int T, int K, const double *x0, const double *v0, double *ck_x, double *ck_v,
                 int n_rec, const int *rec_t, double *rec_x, double *rec_v, double *xT, double *vT) {
    const size_t S = (size_t)m->N * 3, ES = S * m->E;
    double *xa = dup_d(x0, ES), *va = dup_d(v0, ES), *xb = zeros_d(ES), *vb = zeros_d(ES);
    int jr = 0;
    for (int t = 0; t <= T; t++) {
        if (t < T && t % K == 0 && ck_x) { memcpy(ck_x + (size_t)(t / K) * ES, xa, sizeof(double) * ES); memcpy(ck_v + (size_t)(t / K) * ES, va, sizeof(double) * ES); }
        while (jr < n_rec && rec_t[jr] == t) {
            if (rec_x) memcpy(rec_x + (size_t)jr * ES, xa, sizeof(double) * ES);
            if (rec_v) memcpy(rec_v + (size_t)jr * ES, va, sizeof(double) * ES);
            jr++;
        }
        if (t == T) break;
        act_load(m, t);
        orc_step(m, xa, va, xb, vb);
        double *tmp = xa; xa = xb; xb = tmp; tmp = va; va = vb; vb = tmp;
    }
    if (xT) memcpy(xT, xa, sizeof(double) * ES);
    if (vT) memcpy(vT, va, sizeof(double) * ES);
    free(xa); free(va); free(xb); free(vb);
}

/* Backward through T substeps.  Loss cotangents dL/dx at states after loss_t[j] substeps (sorted ascending,
   1 <= loss_t <= T) in loss_ax [n_loss][E][N][3]; optional dL/dv_T in adj_vT.  For each segment, last to
   first, states inside it are regenerated by forward replay from its checkpoint, then the adjoint substeps
   run.  Output dL/dx0, dL/dv0; parameter gradients accumulate in the model. */
void orc_rollout_backward(orc_model *m, int T, int K, const double *ck_x, const double *ck_v, int n_loss, const int *loss_t,
                          const double *loss_ax, const double *adj_vT, double *adj_x0, double *adj_v0) {
    const size_t S = (size_t)m->N * 3, ES = S * m->E;
    double *bx = zeros_d(ES), *bv = zeros_d(ES), *ax = zeros_d(ES), *av = zeros_d(ES);
    double *seg_x = zeros_d(ES * K), *seg_v = zeros_d(ES * K);
    if (adj_vT) memcpy(bv, adj_vT, sizeof(double) * ES);
    int jl = n_loss - 1;
    int n_ck = (T + K - 1) / K;
    for (int c = n_ck - 1; c >= 0; c--) {
        int t0 = c * K, t1 = t0 + K < T ? t0 + K : T;
        memcpy(seg_x, ck_x + (size_t)c * ES, sizeof(double) * ES);
        memcpy(seg_v, ck_v + (size_t)c * ES, sizeof(double) * ES);
        for (int t = t0; t + 1 < t1; t++) { /* replay: state t+1 from state t */
            act_load(m, t);
            orc_step(m, seg_x + (size_t)(t - t0) * ES, seg_v + (size_t)(t - t0) * ES, seg_x + (size_t)(t + 1 - t0) * ES, seg_v + (size_t)(t + 1 - t0) * ES);
        }
        for (int t = t1 - 1; t >= t0; t--) {
            while (jl >= 0 && loss_t[jl] == t + 1) { /* inject dL/dx_{t+1} */
                const double *la = loss_ax + (size_t)jl * ES;
                for (size_t i = 0; i < ES; i++) bx[i] += la[i];
                jl--;
            }
            act_load(m, t);
            orc_step_adjoint(m, seg_x + (size_t)(t - t0) * ES, seg_v + (size_t)(t - t0) * ES, bx, bv, ax, av);
            act_collect(m, t);
            double *tmp = bx; bx = ax; ax = tmp; tmp = bv; bv = av; av = tmp;
        }
    }
    memcpy(adj_x0, bx, sizeof(double) * ES);
    memcpy(adj_v0, bv, sizeof(double) * ES);
    free(bx); free(bv); free(ax); free(av); free(seg_x); free(seg_v);
}

/* bench.py's single-thread CPU baseline (SURVEY.md 8(d) timing protocol); results do not depend on the thread count */
void orc_set_num_threads(int n) {
#ifdef _OPENMP
    extern void omp_set_num_threads(int);
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}
int orc_num_threads(void) {
#ifdef _OPENMP
    extern int omp_get_max_threads(void);
    return omp_get_max_threads();
#else
    return 1;
#endif
}
