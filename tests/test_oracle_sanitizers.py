"""The oracle under AddressSanitizer + UndefinedBehaviorSanitizer: gs_oracle.c is compiled together
with a small C driver (-fsanitize=address,undefined, OpenMP on) that builds a mixed mesh (tets + triangles + a hinge),
switches every optional term on (activation schedules, lift / drag, gravity), and runs forces, energy, a checkpointed
rollout and its backward pass.  Any heap overflow, use after free, leak or undefined operation makes the driver exit
non-zero.  No GPU."""
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

DRIVER = r"""
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
typedef struct orc_model orc_model;
orc_model *orc_create(int N, int M, int Mt, int Mh, int E, const double *x_rest, const double *mass, const unsigned char *pinned, const int *tets,
                      const double *tet_mu, const double *tet_lambda, const double *tet_damp, const int *tris, const double *tri_mu, const double *tri_lambda,
                      const double *tri_damp, const int *hinges, const double *hinge_kb, const double *gravity, double dt, const double *plane_n,
                      double plane_d, double radius, const double *ke, const double *kd, const double *kf, const double *mu_c);
void orc_destroy(orc_model *m);
int orc_set_params(orc_model *m, int group, const double *v);
int orc_get_grads(const orc_model *m, int group, double *out);
void orc_zero_grads(orc_model *m);
void orc_forces(const orc_model *m, const double *x, const double *v, double *f, int mask);
void orc_energy(const orc_model *m, const double *x, int mask, double *U);
void orc_set_act_schedule(orc_model *m, int n_frames, int stride, const double *tet, const double *hinge);
void orc_get_act_schedule_grads(const orc_model *m, double *g_tet, double *g_hinge);
void orc_rollout(orc_model *m, int T, int K, const double *x0, const double *v0, double *ck_x, double *ck_v, int n_rec, const int *rec_t,
                 double *rec_x, double *rec_v, double *xT, double *vT);
void orc_rollout_backward(orc_model *m, int T, int K, const double *ck_x, const double *ck_v, int n_loss, const int *loss_t, const double *loss_ax,
                          const double *adj_vT, double *adj_x0, double *adj_v0);
enum { N = 8, M = 2, MT = 2, MH = 1, E = 2, T = 37, K = 8, F = 3 };
int main(void) {
    /* two tets sharing a face, and a two-triangle strip with one hinge, hovering just above the ground */
    double x[N * 3] = {0, .01, 0, .1, .01, 0, 0, .11, 0, 0, .01, .1, .1, .11, .1, /* cloth */ .3, .005, 0, .4, .005, 0, .3, .005, .1};
    int tets[M * 4] = {0, 1, 2, 3, 1, 2, 3, 4};
    int tris[MT * 3] = {5, 7, 6, 6, 7, 4};
    int hinges[MH * 4] = {5, 4, 7, 6};
    double mass[E * N], tmu[E * M], tla[E * M], tda[E * M], rmu[E * MT], rla[E * MT], rda[E * MT], kb[MH] = {10};
    unsigned char pinned[N] = {0};
    for (int i = 0; i < E * N; i++) mass[i] = 0.1 + 0.01 * i;
    for (int i = 0; i < E * M; i++) { tmu[i] = 1e4; tla[i] = 2e4; tda[i] = 1; }
    for (int i = 0; i < E * MT; i++) { rmu[i] = 1e3; rla[i] = 1e3; rda[i] = 1; }
    double g[3] = {0, -9.8, 0}, n[3] = {0, 1, 0}, ke[E] = {1e4, 2e4}, kd[E] = {10, 5}, kf[E] = {50, 20}, muc[E] = {.5, .3};
    /* tet 1 may be inverted in this numbering: try, and swap two vertices if the oracle rejects it */
    orc_model *m = orc_create(N, M, MT, MH, E, x, mass, pinned, tets, tmu, tla, tda, tris, rmu, rla, rda, hinges, kb, g, 1.0 / 1920, n, 0, 0, ke, kd, kf, muc);
    if (!m) { int t = tets[6]; tets[6] = tets[7]; tets[7] = t; m = orc_create(N, M, MT, MH, E, x, mass, pinned, tets, tmu, tla, tda, tris, rmu, rla, rda, hinges, kb, g, 1.0 / 1920, n, 0, 0, ke, kd, kf, muc); }
    if (!m) { fprintf(stderr, "mesh rejected\n"); return 2; }
    double air[E] = {30, 20}, wind[3] = {.5, -.2, .3};
    orc_set_params(m, 14, air); orc_set_params(m, 15, air); orc_set_params(m, 16, wind);
    double st[F * E * M], sh[F * E * MH];
    for (int i = 0; i < F * E * M; i++) st[i] = 0.02 * ((i % 5) - 2);
    for (int i = 0; i < F * E * MH; i++) sh[i] = 0.1 * ((i % 3) - 1);
    orc_set_act_schedule(m, F, 9, st, sh);
    double x0[E * N * 3], v0[E * N * 3], f[E * N * 3], U[E];
    for (int e = 0; e < E; e++) for (int i = 0; i < N * 3; i++) { x0[e * N * 3 + i] = x[i]; v0[e * N * 3 + i] = 0.1 * ((i * 7 + e) % 5 - 2); }
    orc_forces(m, x0, v0, f, 15); orc_energy(m, x0, 7, U);
    int n_ck = (T + K - 1) / K, rec_t[2] = {16, T}, loss_t[2] = {16, T};
    double *ck_x = calloc((size_t)n_ck * E * N * 3, sizeof(double)), *ck_v = calloc((size_t)n_ck * E * N * 3, sizeof(double));
    double rec_x[2 * E * N * 3], xT[E * N * 3], vT[E * N * 3], ax0[E * N * 3], av0[E * N * 3], cot[2 * E * N * 3];
    orc_rollout(m, T, K, x0, v0, ck_x, ck_v, 2, rec_t, rec_x, NULL, xT, vT);
    for (int i = 0; i < 2 * E * N * 3; i++) cot[i] = rec_x[i] - 0.01;
    orc_zero_grads(m);
    orc_rollout_backward(m, T, K, ck_x, ck_v, 2, loss_t, cot, NULL, ax0, av0);
    double gt[F * E * M], gh[F * E * MH], out[E * N];
    orc_get_act_schedule_grads(m, gt, gh);
    double s = 0;
    for (int grp = 0; grp <= 15; grp++) { memset(out, 0, sizeof out); if (orc_get_grads(m, grp, out) == 0) for (int i = 0; i < E; i++) s += out[i]; }
    for (int i = 0; i < E * N * 3; i++) s += ax0[i] + av0[i] + xT[i];
    for (int i = 0; i < F * E * M; i++) s += gt[i];
    printf("checksum %.6e\n", s);
    free(ck_x); free(ck_v);
    orc_set_act_schedule(m, 0, 1, NULL, NULL);
    orc_destroy(m);
    return s == s ? 0 : 3;
}
"""


def test_oracle_under_asan_and_ubsan(tmp_path):
    drv = tmp_path / "driver.c"
    drv.write_text(DRIVER)
    exe = tmp_path / "driver"
    cmd = ["gcc", "-O1", "-g", "-std=c99", "-fopenmp", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer",
           "-o", str(exe), str(drv), os.path.join(ROOT, "oracle", "gs_oracle.c"), "-lm"]
    subprocess.check_call(cmd)
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", OMP_NUM_THREADS="4")
    r = subprocess.run([str(exe)], capture_output=True, text=True, env=env, timeout=300)
    sys.stdout.write(r.stdout)
    assert r.returncode == 0, r.stderr[-3000:]
    assert "AddressSanitizer" not in r.stderr and "runtime error" not in r.stderr, r.stderr[-3000:]
    assert "checksum" in r.stdout
