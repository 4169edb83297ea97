// gs_elements.cuh -- per-element / per-particle device functions of the hot path, fp32.
//
//   tet_force / tet_adjoint        stable Neo-Hookean constant-strain tets  PAPER.md:575-581, 659-665; A1, A3
//   tri_force / tri_adjoint        same energy on the 3x2 in-plane F       PAPER.md:584; A4
//   hinge_force / hinge_adjoint    dihedral bending, Bridson directions     PAPER.md:585-586; A5, A6
//   contact_force / contact_adjoint penalty contact + relaxed Coulomb       PAPER.md:596-599, 684-688; A7, A8
//   integrate                       semi-implicit Euler                     PAPER.md:618-619, 763-764 (Listing 1)
//
// Shared by the streaming kernels (gs_stream.cu) and the resident kernels (gs_resident.cu).
// Nothing here is shared with oracle/.
#pragma once
#include "gs_math.cuh"

namespace gs {

// MUFU.RCP, <= 1 ulp, no IEEE slow path: element geometry and invariants only (arguments >= 1 or clamped away from 0);
// never contact (hazard H3)
__device__ __forceinline__ float rcp_fast(float x) {
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

// ------------------------------------------------------------------------------------------ tets
// B = D_m^-1 row-major b[k*3+c], V = rest volume.  F = D_s B: column c of F = sum_k d_k b[k][c].
struct TetKin {
    vec3 f1, f2, f3;  // columns of F
    vec3 c1, c2, c3;  // columns of cof F = dJ/dF
    float Ic, J;
};

__device__ __forceinline__ void mat_cols_times_B(const vec3 &d1, const vec3 &d2, const vec3 &d3, const float *b, vec3 &o1, vec3 &o2, vec3 &o3) {
    o1 = madd(madd(b[0] * d1, b[3], d2), b[6], d3);
    o2 = madd(madd(b[1] * d1, b[4], d2), b[7], d3);
    o3 = madd(madd(b[2] * d1, b[5], d2), b[8], d3);
}
// columns times B^T: o_k = sum_c p_c b[k][c]
__device__ __forceinline__ void mat_cols_times_Bt(const vec3 &p1, const vec3 &p2, const vec3 &p3, const float *b, vec3 &o1, vec3 &o2, vec3 &o3) {
    o1 = madd(madd(b[0] * p1, b[1], p2), b[2], p3);
    o2 = madd(madd(b[3] * p1, b[4], p2), b[5], p3);
    o3 = madd(madd(b[6] * p1, b[7], p2), b[8], p3);
}

__device__ __forceinline__ void tet_kin(const vec3 &x0, const vec3 &x1, const vec3 &x2, const vec3 &x3, const float *b, TetKin &k) {
    // edge vectors first (fp32 hazard H2), then F
    mat_cols_times_B(x1 - x0, x2 - x0, x3 - x0, b, k.f1, k.f2, k.f3);
    k.c1 = cross(k.f2, k.f3);
    k.c2 = cross(k.f3, k.f1);
    k.c3 = cross(k.f1, k.f2);
    k.Ic = dot(k.f1, k.f1) + dot(k.f2, k.f2) + dot(k.f3, k.f3);
    k.J = dot(k.f1, k.c1);
}

// P = mu [s1 F - 3/4 cof F] + lambda (J - 1 - act) cof F + k F sym(F^T Fdot),  s1 = 1 - 1/(I_C + 1)
// act: the per-element actuation of PAPER.md:579 (0 = passive)
// nodal forces H = -V P B^T; f[1..3] = columns of H, f[0] = -(sum)
__device__ __forceinline__ void tet_force(const vec3 x[4], const vec3 v[4], const float *b, float V, float mu, float lam, float kd, float act, vec3 f[4]) {
    TetKin k;
    tet_kin(x[0], x[1], x[2], x[3], b, k);
    vec3 g1, g2, g3;
    mat_cols_times_B(v[1] - v[0], v[2] - v[0], v[3] - v[0], b, g1, g2, g3);
    // -V is folded into the three scalar coefficients, so the columns below are those of -V P
    const float s1 = k.Ic * rcp_fast(k.Ic + 1.0f);
    const float ce = -V * (lam * ((k.J - 1.0f) - act) - 0.75f * mu);  // lambda (J - alpha), alpha = 1 + 3mu/(4 lambda) + act  (A1)
    const float ms = -V * mu * s1;
    const float kv = -V * kd, kh = 0.5f * kv;
    // kv S, S = sym(F^T Fdot)
    const float s11 = kv * dot(k.f1, g1), s22 = kv * dot(k.f2, g2), s33 = kv * dot(k.f3, g3);
    const float s12 = kh * (dot(k.f1, g2) + dot(k.f2, g1));
    const float s13 = kh * (dot(k.f1, g3) + dot(k.f3, g1));
    const float s23 = kh * (dot(k.f2, g3) + dot(k.f3, g2));
    const vec3 p1 = madd(madd(madd(madd(ms * k.f1, ce, k.c1), s11, k.f1), s12, k.f2), s13, k.f3);
    const vec3 p2 = madd(madd(madd(madd(ms * k.f2, ce, k.c2), s12, k.f1), s22, k.f2), s23, k.f3);
    const vec3 p3 = madd(madd(madd(madd(ms * k.f3, ce, k.c3), s13, k.f1), s23, k.f2), s33, k.f3);
    mat_cols_times_Bt(p1, p2, p3, b, f[1], f[2], f[3]);
    f[0] = -(f[1] + f[2] + f[3]);
}

// VJP: a[k] = dL/df_k.  Outputs ax[k] = dL/dx_k, av[k] = dL/dv_k contributions (overwritten) and the
// parameter gradients of this element for this substep.
// Everything downstream of A = adj_P = -V G B is linear in A, so the kernel works with A' = G B and folds -V into the
// scalar coefficients; F:A = tr(F^T A) and (F S):A = S:sym(F^T A) reuse the entries of N = sym(F^T A').
// gact = dL/d(act) of this substep: dP/d(act) = -lambda cof F
__device__ __forceinline__ void tet_adjoint(const vec3 x[4], const vec3 v[4], const vec3 a[4], const float *b, float V, float mu, float lam, float kd, float act,
                                            vec3 ax[4], vec3 av[4], float &gmu, float &glam, float &gk, float &gact) {
    TetKin k;
    tet_kin(x[0], x[1], x[2], x[3], b, k);
    vec3 g1, g2, g3;
    mat_cols_times_B(v[1] - v[0], v[2] - v[0], v[3] - v[0], b, g1, g2, g3);
    vec3 A1, A2, A3;  // A' = G B, G = [a1-a0, a2-a0, a3-a0]
    mat_cols_times_B(a[1] - a[0], a[2] - a[0], a[3] - a[0], b, A1, A2, A3);
    const float ip1 = 1.0f / (k.Ic + 1.0f);
    const float s1 = k.Ic * ip1;
    // S = sym(F^T Fdot), N = sym(F^T A')
    const float s11 = dot(k.f1, g1), s22 = dot(k.f2, g2), s33 = dot(k.f3, g3);
    const float s12 = 0.5f * (dot(k.f1, g2) + dot(k.f2, g1));
    const float s13 = 0.5f * (dot(k.f1, g3) + dot(k.f3, g1));
    const float s23 = 0.5f * (dot(k.f2, g3) + dot(k.f3, g2));
    const float n11 = dot(k.f1, A1), n22 = dot(k.f2, A2), n33 = dot(k.f3, A3);
    const float n12 = 0.5f * (dot(k.f1, A2) + dot(k.f2, A1));
    const float n13 = 0.5f * (dot(k.f1, A3) + dot(k.f3, A1));
    const float n23 = 0.5f * (dot(k.f2, A3) + dot(k.f3, A2));
    const float FA = n11 + n22 + n33;
    const float CA = dot(k.c1, A1) + dot(k.c2, A2) + dot(k.c3, A3);
    const float SN = fmaf(s11, n11, fmaf(s22, n22, s33 * n33)) + 2.0f * fmaf(s12, n12, fmaf(s13, n13, s23 * n23));
    // parameter gradients: P is linear in mu, lambda, k
    const float mV = -V;
    const float Jm = (k.J - 1.0f) - act;
    gmu = mV * (s1 * FA - 0.75f * CA);
    glam = mV * (Jm * CA);
    gk = mV * SN;
    gact = V * lam * CA;
    // adj_F = mu s1 A + 2 mu (F:A)/(Ic+1)^2 F + lambda (cof:A) cof + lambda (J - alpha) Dcof[A] + k (A S + Fdot N),  A = -V A'
    const float ms = mV * mu * s1, q = mV * 2.0f * mu * FA * ip1 * ip1, lc = mV * lam * CA, ce = mV * (lam * Jm - 0.75f * mu);
    const float kv = mV * kd;
    const float t11 = kv * s11, t22 = kv * s22, t33 = kv * s33, t12 = kv * s12, t13 = kv * s13, t23 = kv * s23;  // kv S
    const float m11 = kv * n11, m22 = kv * n22, m33 = kv * n33, m12 = kv * n12, m13 = kv * n13, m23 = kv * n23;  // kv N
    const vec3 D1 = cross(A2, k.f3) + cross(k.f2, A3);
    const vec3 D2 = cross(A3, k.f1) + cross(k.f3, A1);
    const vec3 D3 = cross(A1, k.f2) + cross(k.f1, A2);
    vec3 aF1 = madd(madd(madd(ms * A1, q, k.f1), lc, k.c1), ce, D1);
    vec3 aF2 = madd(madd(madd(ms * A2, q, k.f2), lc, k.c2), ce, D2);
    vec3 aF3 = madd(madd(madd(ms * A3, q, k.f3), lc, k.c3), ce, D3);
    aF1 = madd(madd(madd(madd(madd(madd(aF1, t11, A1), t12, A2), t13, A3), m11, g1), m12, g2), m13, g3);
    aF2 = madd(madd(madd(madd(madd(madd(aF2, t12, A1), t22, A2), t23, A3), m12, g1), m22, g2), m23, g3);
    aF3 = madd(madd(madd(madd(madd(madd(aF3, t13, A1), t23, A2), t33, A3), m13, g1), m23, g2), m33, g3);
    const vec3 aG1 = madd(madd(m11 * k.f1, m12, k.f2), m13, k.f3);
    const vec3 aG2 = madd(madd(m12 * k.f1, m22, k.f2), m23, k.f3);
    const vec3 aG3 = madd(madd(m13 * k.f1, m23, k.f2), m33, k.f3);
    // adj_Ds = adj_F B^T
    mat_cols_times_Bt(aF1, aF2, aF3, b, ax[1], ax[2], ax[3]);
    ax[0] = -(ax[1] + ax[2] + ax[3]);
    mat_cols_times_Bt(aG1, aG2, aG3, b, av[1], av[2], av[3]);
    av[0] = -(av[1] + av[2] + av[3]);
}

// ------------------------------------------------------------------------------------------ triangles
// 2x2 B row-major b[0..3], A = rest area.  F (3x2) columns f1 = e1 b00 + e2 b10, f2 = e1 b01 + e2 b11.
__device__ __forceinline__ void tri_force(const vec3 x[3], const vec3 v[3], const float *b, float A, float mu, float lam, float kd, vec3 f[3]) {
    const vec3 e1 = x[1] - x[0], e2 = x[2] - x[0], w1 = v[1] - v[0], w2 = v[2] - v[0];
    const vec3 f1 = madd(b[0] * e1, b[2], e2), f2 = madd(b[1] * e1, b[3], e2);
    const vec3 g1 = madd(b[0] * w1, b[2], w2), g2 = madd(b[1] * w1, b[3], w2);
    const float Ic = dot(f1, f1) + dot(f2, f2);
    const vec3 c = cross(f1, f2);
    const float J = sqrtf(dot(c, c));
    const vec3 n = rcp_fast(fmaxf(J, 1e-12f)) * c;
    const vec3 j1 = cross(f2, n), j2 = cross(n, f1);  // dJ/dF
    // -A (rest area) is folded into the scalar coefficients: p1, p2 are the columns of -A P
    const float ms = -A * mu * Ic * rcp_fast(Ic + 1.0f);
    const float ce = -A * (lam * (J - 1.0f) - (2.0f / 3.0f) * mu);  // lambda (J - alpha2), alpha2 = 1 + 2mu/(3 lambda)  (A4)
    const float kv = -A * kd;
    const float s11 = kv * dot(f1, g1), s22 = kv * dot(f2, g2), s12 = 0.5f * kv * (dot(f1, g2) + dot(f2, g1));
    const vec3 p1 = madd(madd(madd(ms * f1, ce, j1), s11, f1), s12, f2);
    const vec3 p2 = madd(madd(madd(ms * f2, ce, j2), s12, f1), s22, f2);
    f[1] = madd(b[0] * p1, b[1], p2);
    f[2] = madd(b[2] * p1, b[3], p2);
    f[0] = -(f[1] + f[2]);
}

__device__ __forceinline__ void tri_adjoint(const vec3 x[3], const vec3 v[3], const vec3 a[3], const float *b, float A, float mu, float lam, float kd,
                                            vec3 ax[3], vec3 av[3], float &gmu, float &glam, float &gk) {
    const vec3 e1 = x[1] - x[0], e2 = x[2] - x[0], w1 = v[1] - v[0], w2 = v[2] - v[0];
    const vec3 f1 = madd(b[0] * e1, b[2], e2), f2 = madd(b[1] * e1, b[3], e2);
    const vec3 g1 = madd(b[0] * w1, b[2], w2), g2 = madd(b[1] * w1, b[3], w2);
    const vec3 G1 = a[1] - a[0], G2 = a[2] - a[0];
    // A' = G B; the rest area is folded into the scalar coefficients (everything below is linear in adj_P = -A A')
    const vec3 A1 = madd(b[0] * G1, b[2], G2), A2 = madd(b[1] * G1, b[3], G2);
    const float Ic = dot(f1, f1) + dot(f2, f2);
    const vec3 c = cross(f1, f2);
    const float J = sqrtf(dot(c, c));
    const float iJ = rcp_fast(fmaxf(J, 1e-12f));
    const vec3 n = iJ * c;
    const vec3 j1 = cross(f2, n), j2 = cross(n, f1);
    const float ip1 = rcp_fast(Ic + 1.0f), s1 = Ic * ip1;
    const float s11 = dot(f1, g1), s22 = dot(f2, g2), s12 = 0.5f * (dot(f1, g2) + dot(f2, g1));
    const float n11 = dot(f1, A1), n22 = dot(f2, A2), n12 = 0.5f * (dot(f1, A2) + dot(f2, A1));
    const float FA = n11 + n22, JA = dot(j1, A1) + dot(j2, A2);
    const float mA = -A;
    gmu = mA * (s1 * FA - (2.0f / 3.0f) * JA);
    glam = mA * ((J - 1.0f) * JA);
    gk = mA * (fmaf(s11, n11, s22 * n22) + 2.0f * s12 * n12);
    // D(dJ/dF)[A] = [A2 x n + f2 x dn, dn x f1 + n x A1], dc = A1 x f2 + f1 x A2, dn = (dc - n (n.dc))/J
    const vec3 dc = cross(A1, f2) + cross(f1, A2);
    const vec3 dn = iJ * (dc - dot(n, dc) * n);
    const vec3 D1 = cross(A2, n) + cross(f2, dn), D2 = cross(dn, f1) + cross(n, A1);
    const float ms = mA * mu * s1, q = mA * 2.0f * mu * FA * ip1 * ip1, lj = mA * lam * JA, ce = mA * (lam * (J - 1.0f) - (2.0f / 3.0f) * mu);
    const float kv = mA * kd;
    const float t11 = kv * s11, t22 = kv * s22, t12 = kv * s12, m11 = kv * n11, m22 = kv * n22, m12 = kv * n12;
    vec3 aF1 = madd(madd(madd(ms * A1, q, f1), lj, j1), ce, D1);
    vec3 aF2 = madd(madd(madd(ms * A2, q, f2), lj, j2), ce, D2);
    aF1 = madd(madd(madd(madd(aF1, t11, A1), t12, A2), m11, g1), m12, g2);
    aF2 = madd(madd(madd(madd(aF2, t12, A1), t22, A2), m12, g1), m22, g2);
    const vec3 aG1 = madd(m11 * f1, m12, f2), aG2 = madd(m12 * f1, m22, f2);
    ax[1] = madd(b[0] * aF1, b[1], aF2); ax[2] = madd(b[2] * aF1, b[3], aF2); ax[0] = -(ax[1] + ax[2]);
    av[1] = madd(b[0] * aG1, b[1], aG2); av[2] = madd(b[2] * aG1, b[3], aG2); av[0] = -(av[1] + av[2]);
}

// ------------------------------------------------------------------------------------------ lift / drag on triangles
// PAPER.md:586 ("a lift/drag model that approximates the effect of the surrounding air on the surface of mesh"); DESIGN.md
// A21: F = -A s (k_drag vb + k_lift (n.vb) n), c = (x1-x0) x (x2-x0), A = |c|/2, n = c/|c|, vb = mean vertex velocity -
// wind, s = sqrt(|vb|^2 + eps^2); a third of F on each vertex.  Written with L = |c|, u = c.vb: F = -(s/2) (k_drag L vb + k_lift u c / L).
constexpr float kAeroEps2 = 1e-12f;  // (1e-6 m/s)^2
__device__ __forceinline__ void aero_force_add(const vec3 x[3], const vec3 v[3], const vec3 &wind, float kdrag, float klift, vec3 f[3]) {
    const vec3 e1 = x[1] - x[0], e2 = x[2] - x[0];
    const vec3 c = cross(e1, e2);
    const vec3 vb = (1.0f / 3.0f) * (v[0] + v[1] + v[2]) - wind;
    const float L2 = dot(c, c), iL = rsqrtf(L2), L = L2 * iL;
    const float s = sqrtf(dot(vb, vb) + kAeroEps2), u = dot(c, vb);
    const vec3 F3 = (-s * (1.0f / 6.0f)) * madd((kdrag * L) * vb, klift * u * iL, c);  // F / 3
    f[0] += F3; f[1] += F3; f[2] += F3;
}
// VJP (a_k = dL/df_k): adds to ax, av; gd, gl = this substep's dL/dk_drag, dL/dk_lift of the triangle.  With ab = mean a_k,
// P = k_drag L vb + k_lift u c / L:  dL/dvb = -(ab.P)/(2s) vb - (s/2) k_drag L ab - (s/2) k_lift (ab.c)/L c;
// dL/dc = -(s/2) k_drag (ab.vb) n - (s/2) k_lift [(ab.c)/L vb + (u/L) ab - u (ab.c)/L^2 n]; dL/de1 = e2 x dL/dc, dL/de2 = dL/dc x e1
__device__ __forceinline__ void aero_adjoint_add(const vec3 x[3], const vec3 v[3], const vec3 a[3], const vec3 &wind, float kdrag, float klift,
                                                 vec3 ax[3], vec3 av[3], float &gd, float &gl) {
    const vec3 e1 = x[1] - x[0], e2 = x[2] - x[0];
    const vec3 c = cross(e1, e2);
    const vec3 vb = (1.0f / 3.0f) * (v[0] + v[1] + v[2]) - wind;
    const vec3 ab = (1.0f / 3.0f) * (a[0] + a[1] + a[2]);
    const float L2 = dot(c, c), iL = rsqrtf(L2), L = L2 * iL;
    const vec3 n = iL * c;
    const float s = sqrtf(dot(vb, vb) + kAeroEps2), hs = 0.5f * s, u = dot(c, vb), ac = dot(ab, c), avb = dot(ab, vb);
    gd = -hs * L * avb;
    gl = -hs * u * ac * iL;
    const float aP = kdrag * L * avb + klift * u * iL * ac;
    const vec3 gv = (1.0f / 3.0f) * madd(madd((-0.5f * aP / s) * vb, -hs * kdrag * L, ab), -hs * klift * ac * iL, c);
    const vec3 gc = madd((-hs * kdrag * avb) * n, -hs * klift, madd(madd((ac * iL) * vb, u * iL, ab), -u * ac * iL * iL, n));
    const vec3 t1 = cross(e2, gc), t2 = cross(gc, e1);
    ax[1] += t1; ax[2] += t2; ax[0] -= t1 + t2;
    av[0] += gv; av[1] += gv; av[2] += gv;
}

// ------------------------------------------------------------------------------------------ hinges
// vertices: x[0], x[1] wings; x[2], x[3] the shared edge.  theta = signed dihedral (0 when flat);
// f_i = k_b l0 sin((theta - theta0)/2 + alpha) d_i, d_i = -d(theta)/dx_i (Bridson directions), alpha the per-edge actuation.
// Rest constants per hinge: s0h = sin(theta0/2), c0h = cos(theta0/2), kl = k_b * l0 (fp64 on the host).
struct HingeGeo {
    vec3 p13, p14, p23, p24, n1, n2, eh, m1, m2;
    float L, iL, i1, i2, c13, c14, c23, c24, sh, ch;  // sh, ch = sin, cos of (theta - theta0)/2
};
// sa, ca = sin, cos of the per-edge actuation alpha (sin(phi/2 + alpha)); (0, 1) = passive
__device__ __forceinline__ void hinge_geo(const vec3 x[4], float s0h, float c0h, float sa, float ca, HingeGeo &h) {
    h.p13 = x[0] - x[2]; h.p14 = x[0] - x[3]; h.p23 = x[1] - x[2]; h.p24 = x[1] - x[3];
    h.n1 = cross(h.p13, h.p14); h.n2 = cross(h.p24, h.p23);
    const vec3 e = x[3] - x[2];
    const float L2 = dot(e, e);
    h.iL = rsqrtf(L2);
    h.L = L2 * h.iL;
    h.eh = h.iL * e;
    const float n1s = dot(h.n1, h.n1), n2s = dot(h.n2, h.n2);
    h.i1 = rcp_fast(n1s); h.i2 = rcp_fast(n2s);
    h.m1 = h.i1 * h.n1; h.m2 = h.i2 * h.n2;
    h.c13 = dot(h.p13, h.eh); h.c14 = dot(h.p14, h.eh); h.c23 = dot(h.p23, h.eh); h.c24 = dot(h.p24, h.eh);
    // (sin, cos) of theta, then the half angle by the branch that does not cancel (hazard H1: never
    // sqrt((1 - cos theta)/2) near theta = 0, where flat cloth lives), then the rest-angle shift -- no atan2 / sin
    const float inv = rsqrtf(n1s * n2s);
    const float sn = dot(cross(h.n1, h.n2), h.eh) * inv, cs = dot(h.n1, h.n2) * inv;
    float sht, cht;
    if (cs >= 0.0f) {
        cht = sqrtf(0.5f * (1.0f + cs));
        sht = 0.5f * sn * rcp_fast(cht);
    } else {
        const float a = sqrtf(0.5f * (1.0f - cs));
        sht = copysignf(a, sn);
        cht = 0.5f * fabsf(sn) * rcp_fast(a);
    }
    const float s1 = sht * c0h - cht * s0h, c1 = cht * c0h + sht * s0h;  // (theta - theta0)/2
    h.sh = s1 * ca + c1 * sa;
    h.ch = c1 * ca - s1 * sa;
}
__device__ __forceinline__ void hinge_dirs(const HingeGeo &h, vec3 d[4]) {
    d[0] = h.L * h.m1;
    d[1] = h.L * h.m2;
    d[2] = madd(h.c14 * h.m1, h.c24, h.m2);
    d[3] = -madd(h.c13 * h.m1, h.c23, h.m2);
}
__device__ __forceinline__ void hinge_force(const vec3 x[4], float s0h, float c0h, float kl, float sa, float ca, vec3 f[4]) {
    HingeGeo h;
    hinge_geo(x, s0h, c0h, sa, ca, h);
    vec3 d[4];
    hinge_dirs(h, d);
    const float s = kl * h.sh;
    f[0] = s * d[0]; f[1] = s * d[1]; f[2] = s * d[2]; f[3] = s * d[3];
}
// VJP = JVP (the force is conservative): ax_j = -E'' s d_j + E' Dd_j[a], s = sum_i d_i . a_i
// gkb = dL/dk_b of this substep: the force is linear in k_b, dL/dk_b = l0 sin((theta - theta0)/2) sum_i d_i . a_i
// gact = dL/d(alpha) of this substep = k_b l0 cos(ph) s (and dL/d(theta0) = -gact / 2: theta0 enters the same argument as -theta0/2)
__device__ __forceinline__ void hinge_adjoint(const vec3 x[4], const vec3 a[4], float s0h, float c0h, float kl, float l0, float sa, float ca, vec3 ax[4],
                                              float &gkb, float &gact) {
    HingeGeo h;
    hinge_geo(x, s0h, c0h, sa, ca, h);
    vec3 d[4];
    hinge_dirs(h, d);
    const vec3 q13 = a[0] - a[2], q14 = a[0] - a[3], q23 = a[1] - a[2], q24 = a[1] - a[3];
    const vec3 dn1 = cross(q13, h.p14) + cross(h.p13, q14);
    const vec3 dn2 = cross(q24, h.p23) + cross(h.p24, q23);
    const vec3 de = a[3] - a[2];
    const float dL = dot(h.eh, de);
    const vec3 deh = h.iL * (de - dL * h.eh);
    const vec3 dm1 = h.i1 * (dn1 - (2.0f * dot(h.n1, dn1) * h.i1) * h.n1);
    const vec3 dm2 = h.i2 * (dn2 - (2.0f * dot(h.n2, dn2) * h.i2) * h.n2);
    const float dc13 = dot(q13, h.eh) + dot(h.p13, deh), dc14 = dot(q14, h.eh) + dot(h.p14, deh);
    const float dc23 = dot(q23, h.eh) + dot(h.p23, deh), dc24 = dot(q24, h.eh) + dot(h.p24, deh);
    // s = sum_i d_i . a_i written with cotangent differences only (sum_i d_i = 0): the adjoint field is smooth,
    // so the plain sum cancels to ~1e-4 of its terms and would lose that many digits in fp32
    const float s = dot(h.m1, h.c13 * q14 - h.c14 * q13) + dot(h.m2, h.c23 * q24 - h.c24 * q23);
    const float E1 = kl * h.sh, E2s = 0.5f * kl * h.ch * s;
    gkb = l0 * h.sh * s;
    gact = 2.0f * E2s;
    ax[0] = madd(-E2s * d[0], E1, madd(dL * h.m1, h.L, dm1));
    ax[1] = madd(-E2s * d[1], E1, madd(dL * h.m2, h.L, dm2));
    ax[2] = madd(-E2s * d[2], E1, madd(madd(madd(dc14 * h.m1, h.c14, dm1), dc24, h.m2), h.c24, dm2));
    ax[3] = madd(-E2s * d[3], -E1, madd(madd(madd(dc13 * h.m1, h.c13, dm1), dc23, h.m2), h.c23, dm2));
}

// ------------------------------------------------------------------------------------------ contact
struct ContactParams {
    vec3 n;
    float d, r, ke, kd, kf, mu;
};
// f_n = -ke c - kd min(v_n, 0) (>= 0), f_f = -v_t min(kf, mu f_n / |v_t|); true divisions (hazard H3)
__device__ __forceinline__ vec3 contact_force(const ContactParams &cp, const vec3 &x, const vec3 &v) {
    const float c = dot(cp.n, x) - cp.d - cp.r;
    if (!(c < 0.0f)) return zero3();
    const float vn = dot(cp.n, v);
    const float fn = -cp.ke * c - cp.kd * fminf(vn, 0.0f);
    const vec3 vt = v - vn * cp.n;
    const float s = sqrtf(dot(vt, vt));
    const float coef = fminf(cp.kf, __fdiv_rn(cp.mu * fn, fmaxf(s, 1e-12f)));
    return fn * cp.n - coef * vt;
}
// a = dL/df; adds the contact VJP to ax, av.  gp[4] = this particle's contributions to dL/dk_e, dL/dk_d, dL/dk_f,
// dL/dmu_c (zero when not in contact): with a.f = f_n afn, d/dk_e = -c afn, d/dk_d = -min(v_n, 0) afn;
// stick: d/dk_f = -(v_t.a_t); slip: d/dmu_c = -f_n (v_t.a_t)/s
__device__ __forceinline__ void contact_adjoint(const ContactParams &cp, const vec3 &x, const vec3 &v, const vec3 &a, vec3 &ax, vec3 &av, float gp[4]) {
    gp[0] = gp[1] = gp[2] = gp[3] = 0.0f;
    const float c = dot(cp.n, x) - cp.d - cp.r;
    if (!(c < 0.0f)) return;
    const float vn = dot(cp.n, v);
    const float fn = -cp.ke * c - cp.kd * fminf(vn, 0.0f);
    const vec3 vt = v - vn * cp.n;
    const float s = sqrtf(dot(vt, vt)), sg = fmaxf(s, 1e-12f);
    const float na = dot(cp.n, a);
    const vec3 at = a - na * cp.n;
    const float vta = dot(vt, at);
    float afn;
    vec3 avt;
    if (__fdiv_rn(cp.mu * fn, sg) >= cp.kf) {  // stick
        afn = na;
        avt = -cp.kf * at;
        gp[2] = -vta;
    } else {  // slip
        const float is = __fdiv_rn(1.0f, sg);
        afn = na - cp.mu * vta * is;
        avt = (-cp.mu * fn * is) * (at - (vta * is * is) * vt);
        gp[3] = -fn * vta * is;
    }
    gp[0] = -c * afn;
    gp[1] = -fminf(vn, 0.0f) * afn;
    av += avt;
    ax += (-cp.ke * afn) * cp.n;
    if (vn < 0.0f) av += (-cp.kd * afn) * cp.n;
}

// ------------------------------------------------------------------------------------------ integrate
// Listing 1: v1 = v0 + (f0 w + g step(w)) dt ; x1 = x0 + v1 dt
__device__ __forceinline__ void integrate(const vec3 &x, const vec3 &v, const vec3 &f, float w, const vec3 &g, float dt, vec3 &x1, vec3 &v1) {
    const float on = w > 0.0f ? 1.0f : 0.0f;
    v1 = madd(v, dt, madd(on * g, w, f));
    x1 = madd(x, dt, v1);
}

}  // namespace gs
