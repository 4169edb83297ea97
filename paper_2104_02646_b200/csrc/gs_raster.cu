// gs_raster.cu -- soft silhouette rasteriser on a headless device buffer and its adjoint.
//
// PAPER.md:168-172 (section 2.2): the renderers "replace discontinuous triangle mesh edges with smooth sigmoids ... blurring
// triangle edges into semi-transparent boundaries".  The paper prints no formula; reading A22 takes the SoftRas
// silhouette as SPEC.md:251 states it:
//     D_j(p) = sigmoid(delta_j(p) d^2(p, boundary of triangle j) / sigma),  delta = +1 inside, -1 outside (NDC distances)
//     S(p)   = 1 - prod_j (1 - D_j(p));     loss ("pixelwise MSE")  L = scale sum_p (S(p) - S*(p))^2
// Camera: pinhole, p_cam = R x + t, drawn iff z_cam > near for all three vertices, NDC (u, v) = (fx X / Z, fy Y / Z), pixel
// (i, j) centre at u = 2 (i + 1/2) / W - 1, v = 2 (j + 1/2) / H - 1.  The colour channel (A22b) is in the second half of this file.
//
// Kernels (plain fp32 ALU work, no tensor cores: per pixel x per triangle distance evaluations):
//   k_rs_project      particles -> NDC
//   k_rs_pack         per (environment, triangle): the three NDC vertices + the bounding box grown by the radius beyond which
//                     an outside pixel's D is below fp32 resolution of 1 - D (d^2 > 40 sigma: D < 5e-18)
//   k_rs_forward      one CTA per 16 x 16 pixel tile: triangles are staged 256 at a time, culled against the tile with a
//                     ballot compaction, every thread folds the survivors into its pixel's product; writes S and, when a
//                     target is given, the block-reduced loss
//   k_rs_backward     same walk, twice: the pixel's full product first, then per surviving triangle
//                     dL/ds = dL/dS prod_{i != j}(1 - D_i) D_j (1 - D_j) / sigma = dL/dS keep D_j / sigma (no division), the
//                     closest-edge weights, a warp shuffle reduction of the six vertex components and one atomicAdd per
//                     component and warp
//   k_rs_project_adj  dL/d(NDC) -> dL/dx through the projection Jacobian
// Nothing here is shared with oracle/raster_oracle.py.
#include <cstdint>

#include "gs_internal.h"

namespace gs {

struct CamDev {
    float R[9], t[3], fx, fy, sigma, near_z, inv_sigma, cull_r;
    int W, H;
};

constexpr int kRsTile = 16;            // pixels per tile side; 256 threads per CTA
constexpr int kRsChunk = 256;          // triangles staged per round
constexpr float kRsCull = 40.0f;       // outside pixels with d^2 > kRsCull * sigma contribute D < exp(-40)

__global__ void k_rs_project(CamDev cam, int E, int N, const float *__restrict__ x, float4 *__restrict__ ndc) {
    const size_t total = (size_t)E * N;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        const float px = x[3 * i], py = x[3 * i + 1], pz = x[3 * i + 2];
        const float X = cam.R[0] * px + cam.R[1] * py + cam.R[2] * pz + cam.t[0];
        const float Y = cam.R[3] * px + cam.R[4] * py + cam.R[5] * pz + cam.t[1];
        const float Z = cam.R[6] * px + cam.R[7] * py + cam.R[8] * pz + cam.t[2];
        const bool vis = Z > cam.near_z;
        const float iz = vis ? 1.0f / Z : 0.0f;
        ndc[i] = make_float4(cam.fx * X * iz, cam.fy * Y * iz, Z, vis ? 1.0f : 0.0f);
    }
}

// tri record: a = (u0, v0, u1, v1), b = (u2, v2, drawn, 0), box = (umin, vmin, umax, vmax) grown by cull_r
struct TriRec { float4 a, b, box; };

__global__ void k_rs_pack(CamDev cam, int E, int N, int Mt, const int *__restrict__ tris, const float4 *__restrict__ ndc, TriRec *__restrict__ rec) {
    const size_t total = (size_t)E * Mt;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        const int env = (int)(i / Mt), j = (int)(i - (size_t)env * Mt);
        const float4 p0 = ndc[(size_t)env * N + tris[3 * j]], p1 = ndc[(size_t)env * N + tris[3 * j + 1]], p2 = ndc[(size_t)env * N + tris[3 * j + 2]];
        const bool drawn = p0.w > 0.f && p1.w > 0.f && p2.w > 0.f;
        TriRec r;
        r.a = make_float4(p0.x, p0.y, p1.x, p1.y);
        r.b = make_float4(p2.x, p2.y, drawn ? 1.0f : 0.0f, 0.f);
        const float m = cam.cull_r;
        r.box = drawn ? make_float4(fminf(p0.x, fminf(p1.x, p2.x)) - m, fminf(p0.y, fminf(p1.y, p2.y)) - m, fmaxf(p0.x, fmaxf(p1.x, p2.x)) + m,
                                    fmaxf(p0.y, fmaxf(p1.y, p2.y)) + m)
                      : make_float4(1e30f, 1e30f, -1e30f, -1e30f);
        rec[i] = r;
    }
}

// squared distance of p to segment ab, closest-point parameter and offset p - c
__device__ __forceinline__ float seg_d2(float pu, float pv, float au, float av, float bu, float bv, float &t, float &du, float &dv) {
    const float eu = bu - au, ev = bv - av, den = eu * eu + ev * ev;
    t = den > 0.f ? fminf(fmaxf(__fdiv_rn((pu - au) * eu + (pv - av) * ev, den), 0.f), 1.f) : 0.f;
    du = pu - (au + t * eu); dv = pv - (av + t * ev);
    return du * du + dv * dv;
}
// signed squared distance s = delta d^2 of pixel p to triangle (a, b); k = closest edge (k -> k+1), t, du, dv of it
__device__ __forceinline__ float tri_signed_d2(float pu, float pv, const float4 &a, const float4 &b, int &k, float &t, float &du, float &dv) {
    float t1, du1, dv1, t2, du2, dv2;
    float d = seg_d2(pu, pv, a.x, a.y, a.z, a.w, t, du, dv);
    k = 0;
    const float d1 = seg_d2(pu, pv, a.z, a.w, b.x, b.y, t1, du1, dv1);
    if (d1 < d) { d = d1; k = 1; t = t1; du = du1; dv = dv1; }
    const float d2 = seg_d2(pu, pv, b.x, b.y, a.x, a.y, t2, du2, dv2);
    if (d2 < d) { d = d2; k = 2; t = t2; du = du2; dv = dv2; }
    const float e0 = (a.z - a.x) * (pv - a.y) - (a.w - a.y) * (pu - a.x);
    const float e1 = (b.x - a.z) * (pv - a.w) - (b.y - a.w) * (pu - a.z);
    const float e2 = (a.x - b.x) * (pv - b.y) - (a.y - b.y) * (pu - b.x);
    const bool inside = (e0 > 0.f && e1 > 0.f && e2 > 0.f) || (e0 < 0.f && e1 < 0.f && e2 < 0.f);
    return inside ? d : -d;
}
__device__ __forceinline__ float sigmoidf_(float a) { return 0.5f * (1.0f + tanhf(0.5f * a)); }

// stage up to kRsChunk triangle records of this round, keep those whose grown box meets the tile: returns the count
__device__ __forceinline__ int stage_tris(const TriRec *__restrict__ rec, int j0, int Mt, float tu0, float tv0, float tu1, float tv1, float4 *sa, float4 *sb,
                                          int *sj, int *s_cnt) {
    const int tid = threadIdx.y * kRsTile + threadIdx.x, j = j0 + tid;
    if (tid == 0) *s_cnt = 0;
    __syncthreads();
    bool hit = false;
    TriRec r;
    if (j < Mt) {
        r = rec[j];
        hit = r.b.z > 0.f && r.box.x <= tu1 && r.box.z >= tu0 && r.box.y <= tv1 && r.box.w >= tv0;
    }
    const unsigned m = __ballot_sync(0xffffffffu, hit);
    int base = 0;
    if ((tid & 31) == 0 && m) base = atomicAdd(s_cnt, __popc(m));
    base = __shfl_sync(0xffffffffu, base, 0);
    if (hit) {
        const int o = base + __popc(m & ((1u << (tid & 31)) - 1u));
        sa[o] = r.a; sb[o] = r.b; sj[o] = j;
    }
    __syncthreads();
    return *s_cnt;
}

// grid (tiles_x, tiles_y, E).  image [E][H][W] out (may be null); target [E][H][W] / loss [E] (atomicAdd) optional.
__global__ void __launch_bounds__(kRsTile *kRsTile) k_rs_forward(CamDev cam, int Mt, const TriRec *__restrict__ rec, float *__restrict__ image,
                                                                  const float *__restrict__ target, float scale, float *__restrict__ loss) {
    __shared__ float4 sa[kRsChunk], sb[kRsChunk];
    __shared__ int sj[kRsChunk], s_cnt;
    __shared__ float red[8];
    const int env = blockIdx.z, pi = blockIdx.x * kRsTile + threadIdx.x, pj = blockIdx.y * kRsTile + threadIdx.y;
    const float su = 2.0f / cam.W, sv = 2.0f / cam.H;
    const float pu = (pi + 0.5f) * su - 1.0f, pv = (pj + 0.5f) * sv - 1.0f;
    const float tu0 = blockIdx.x * kRsTile * su - 1.0f, tv0 = blockIdx.y * kRsTile * sv - 1.0f, tu1 = tu0 + kRsTile * su, tv1 = tv0 + kRsTile * sv;
    const TriRec *re = rec + (size_t)env * Mt;
    float keep = 1.0f;
    for (int j0 = 0; j0 < Mt; j0 += kRsChunk) {
        const int n = stage_tris(re, j0, Mt, tu0, tv0, tu1, tv1, sa, sb, sj, &s_cnt);
        for (int q = 0; q < n; q++) {
            int k; float t, du, dv;
            const float s = tri_signed_d2(pu, pv, sa[q], sb[q], k, t, du, dv);
            keep *= 1.0f - sigmoidf_(s * cam.inv_sigma);
        }
        __syncthreads();
    }
    const bool in = pi < cam.W && pj < cam.H;
    const float S = 1.0f - keep;
    const size_t o = ((size_t)env * cam.H + pj) * cam.W + pi;
    if (in && image) image[o] = S;
    if (target) {
        float d = in ? S - target[o] : 0.f;
        d *= d;
        for (int w = 16; w > 0; w >>= 1) d += __shfl_xor_sync(0xffffffffu, d, w);
        const int tid = threadIdx.y * kRsTile + threadIdx.x;
        if ((tid & 31) == 0) red[tid >> 5] = d;
        __syncthreads();
        if (tid == 0) {
            float tot = 0.f;
            for (int w = 0; w < 8; w++) tot += red[w];
            atomicAdd(loss + env, scale * tot);
        }
    }
}

// dL/d(NDC vertices) of L = scale sum_p (S - S*)^2; g_ndc [E][N] float2, zero on entry
__global__ void __launch_bounds__(kRsTile *kRsTile) k_rs_backward(CamDev cam, int N, int Mt, const int *__restrict__ tris, const TriRec *__restrict__ rec,
                                                                   const float *__restrict__ target, float scale, float2 *__restrict__ g_ndc) {
    __shared__ float4 sa[kRsChunk], sb[kRsChunk];
    __shared__ int sj[kRsChunk], s_cnt;
    const int env = blockIdx.z, pi = blockIdx.x * kRsTile + threadIdx.x, pj = blockIdx.y * kRsTile + threadIdx.y;
    const float su = 2.0f / cam.W, sv = 2.0f / cam.H;
    const float pu = (pi + 0.5f) * su - 1.0f, pv = (pj + 0.5f) * sv - 1.0f;
    const float tu0 = blockIdx.x * kRsTile * su - 1.0f, tv0 = blockIdx.y * kRsTile * sv - 1.0f, tu1 = tu0 + kRsTile * su, tv1 = tv0 + kRsTile * sv;
    const TriRec *re = rec + (size_t)env * Mt;
    const bool in = pi < cam.W && pj < cam.H;
    const int lane = (threadIdx.y * kRsTile + threadIdx.x) & 31;
    // pass 1: the pixel's product over all triangles
    float keep = 1.0f;
    for (int j0 = 0; j0 < Mt; j0 += kRsChunk) {
        const int n = stage_tris(re, j0, Mt, tu0, tv0, tu1, tv1, sa, sb, sj, &s_cnt);
        for (int q = 0; q < n; q++) {
            int k; float t, du, dv;
            keep *= 1.0f - sigmoidf_(tri_signed_d2(pu, pv, sa[q], sb[q], k, t, du, dv) * cam.inv_sigma);
        }
        __syncthreads();
    }
    const size_t o = ((size_t)env * cam.H + pj) * cam.W + pi;
    const float gS = in ? 2.0f * scale * ((1.0f - keep) - target[o]) : 0.f;
    const float gk = gS * keep * cam.inv_sigma;  // dL/ds_j = gS prod_{i != j}(1 - D_i) D_j (1 - D_j) / sigma = gk D_j
    // pass 2: per triangle, closest-edge weights; warp-reduce the six vertex components, one atomic per component and warp
    for (int j0 = 0; j0 < Mt; j0 += kRsChunk) {
        const int n = stage_tris(re, j0, Mt, tu0, tv0, tu1, tv1, sa, sb, sj, &s_cnt);
        for (int q = 0; q < n; q++) {
            int k; float t, du, dv;
            const float s = tri_signed_d2(pu, pv, sa[q], sb[q], k, t, du, dv);
            const float gs = gk * sigmoidf_(s * cam.inv_sigma) * (s >= 0.f ? 1.0f : -1.0f);
            if (!__any_sync(0xffffffffu, gs != 0.f)) continue;
            const float wa = -2.0f * (1.0f - t) * gs, wb = -2.0f * t * gs;
            float c[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};  // (u, v) of vertices 0, 1, 2
            const int ka = k, kb = k == 2 ? 0 : k + 1;
#pragma unroll
            for (int v = 0; v < 3; v++) {
                const float w = (v == ka ? wa : 0.f) + (v == kb ? wb : 0.f);
                c[2 * v] = w * du; c[2 * v + 1] = w * dv;
            }
#pragma unroll
            for (int i = 0; i < 6; i++)
                for (int w = 16; w > 0; w >>= 1) c[i] += __shfl_xor_sync(0xffffffffu, c[i], w);
            if (lane == 0) {
                const int *tr = tris + 3 * (size_t)sj[q];
#pragma unroll
                for (int v = 0; v < 3; v++) {
                    float2 *g = g_ndc + (size_t)env * N + tr[v];
                    if (c[2 * v] != 0.f) atomicAdd(&g->x, c[2 * v]);
                    if (c[2 * v + 1] != 0.f) atomicAdd(&g->y, c[2 * v + 1]);
                }
            }
        }
        __syncthreads();
    }
}

// d(u, v)/d(p_cam) = [[fx / Z, 0, -fx X / Z^2], [0, fy / Z, -fy Y / Z^2]], dp_cam/dx = R
__global__ void k_rs_project_adj(CamDev cam, int E, int N, const float *__restrict__ x, const float2 *__restrict__ g_ndc, float *__restrict__ adj_x) {
    const size_t total = (size_t)E * N;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        const float px = x[3 * i], py = x[3 * i + 1], pz = x[3 * i + 2];
        const float X = cam.R[0] * px + cam.R[1] * py + cam.R[2] * pz + cam.t[0];
        const float Y = cam.R[3] * px + cam.R[4] * py + cam.R[5] * pz + cam.t[1];
        const float Z = cam.R[6] * px + cam.R[7] * py + cam.R[8] * pz + cam.t[2];
        float gx = 0.f, gy = 0.f, gz = 0.f;
        if (Z > cam.near_z) {
            const float2 g = g_ndc[i];
            const float iz = 1.0f / Z;
            gx = g.x * cam.fx * iz; gy = g.y * cam.fy * iz; gz = -(g.x * cam.fx * X + g.y * cam.fy * Y) * iz * iz;
        }
        adj_x[3 * i] = cam.R[0] * gx + cam.R[3] * gy + cam.R[6] * gz;
        adj_x[3 * i + 1] = cam.R[1] * gx + cam.R[4] * gy + cam.R[7] * gz;
        adj_x[3 * i + 2] = cam.R[2] * gx + cam.R[5] * gy + cam.R[8] * gz;
    }
}

// ------------------------------------------------------------------------------------------ colour channel (A22b)
// depth-softmax aggregation of barycentric vertex colours ("only colour" shading):
//   lam_k screen-space barycentrics, w = clip(lam, 0, 1) renormalised, z_j = sum w_k Z_k, zbar_j = (far - z_j) / (far - near),
//   C_j = sum w_k c_k,  I = (sum_j D_j e^{zbar_j / gamma} C_j + e^{eps / gamma} C_b) / (sum_j D_j e^{zbar_j / gamma} + e^{eps / gamma})
// over the drawn triangles with |2 area| > 1e-5 x (longest edge)^2 (no slivers) and s_j(p) >= -40 sigma.  The exponents are taken relative to a running
// maximum m (it cancels in the quotient); images are planar [E][3][H][W].
struct ShadeDev {
    float inv_gamma, eps_g, far_z, inv_range, bg[3], s_cut;
};
struct TriCol { float4 v0, v1, v2; };  // per vertex (Z, r, g, b)

__global__ void k_rs_pack_rgb(int E, int N, int Mt, const int *__restrict__ tris, const float4 *__restrict__ ndc, const float *__restrict__ colour,
                              TriRec *__restrict__ rec, TriCol *__restrict__ col) {
    const size_t total = (size_t)E * Mt;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        const int env = (int)(i / Mt), j = (int)(i - (size_t)env * Mt);
        const size_t i0 = (size_t)env * N + tris[3 * j], i1 = (size_t)env * N + tris[3 * j + 1], i2 = (size_t)env * N + tris[3 * j + 2];
        const float4 p0 = ndc[i0], p1 = ndc[i1], p2 = ndc[i2];
        const float A2 = (p1.x - p0.x) * (p2.y - p0.y) - (p1.y - p0.y) * (p2.x - p0.x);
        const float l01 = (p1.x - p0.x) * (p1.x - p0.x) + (p1.y - p0.y) * (p1.y - p0.y), l12 = (p2.x - p1.x) * (p2.x - p1.x) + (p2.y - p1.y) * (p2.y - p1.y),
                    l20 = (p0.x - p2.x) * (p0.x - p2.x) + (p0.y - p2.y) * (p0.y - p2.y);
        rec[i].b.w = fabsf(A2) > 1e-5f * fmaxf(l01, fmaxf(l12, l20)) ? 1.0f : 0.0f;  // rec[i].a, .box and .b.xyz are k_rs_pack's
        TriCol c;
        c.v0 = make_float4(p0.z, colour[3 * i0], colour[3 * i0 + 1], colour[3 * i0 + 2]);
        c.v1 = make_float4(p1.z, colour[3 * i1], colour[3 * i1 + 1], colour[3 * i1 + 2]);
        c.v2 = make_float4(p2.z, colour[3 * i2], colour[3 * i2 + 1], colour[3 * i2 + 2]);
        col[i] = c;
    }
}

// as stage_tris, with the colour records of the survivors
__device__ __forceinline__ int stage_tris_rgb(const TriRec *__restrict__ rec, const TriCol *__restrict__ col, int j0, int Mt, float tu0, float tv0, float tu1,
                                              float tv1, float4 *sa, float4 *sb, float4 *sc, int *sj, int *s_cnt) {
    const int tid = threadIdx.y * kRsTile + threadIdx.x, j = j0 + tid;
    if (tid == 0) *s_cnt = 0;
    __syncthreads();
    bool hit = false;
    TriRec r;
    if (j < Mt) {
        r = rec[j];
        hit = r.b.z > 0.f && r.b.w > 0.f && r.box.x <= tu1 && r.box.z >= tu0 && r.box.y <= tv1 && r.box.w >= tv0;
    }
    const unsigned m = __ballot_sync(0xffffffffu, hit);
    int base = 0;
    if ((tid & 31) == 0 && m) base = atomicAdd(s_cnt, __popc(m));
    base = __shfl_sync(0xffffffffu, base, 0);
    if (hit) {
        const int o = base + __popc(m & ((1u << (tid & 31)) - 1u));
        const TriCol c = col[j];
        sa[o] = r.a; sb[o] = r.b; sj[o] = j;
        sc[3 * o] = c.v0; sc[3 * o + 1] = c.v1; sc[3 * o + 2] = c.v2;
    }
    __syncthreads();
    return *s_cnt;
}

// one pixel x one triangle of the colour channel
struct RgbTerm {
    float s, D, omD, t, du, dv, lam[3], w[3], isu, iA, e, C[3];  // omD = 1 - D
    int k;
    bool on;
};
__device__ __forceinline__ void rgb_term(const CamDev &cam, const ShadeDev &sh, float pu, float pv, const float4 &a, const float4 &b, const float4 *c, RgbTerm &r) {
    r.s = tri_signed_d2(pu, pv, a, b, r.k, r.t, r.du, r.dv);
    r.on = r.s >= sh.s_cut;
    if (!r.on) return;
    // D multiplies e^{zbar / gamma}: its tail must be accurate in RELATIVE terms (the tanh form of the silhouette rounds
    // D < 6e-8 to zero); s / sigma >= -40 keeps e^{-s / sigma} finite
    const float ex = expf(-r.s * cam.inv_sigma);
    r.D = 1.0f / (1.0f + ex);
    r.omD = ex * r.D;
    const float e0 = (a.z - a.x) * (pv - a.y) - (a.w - a.y) * (pu - a.x);
    const float e1 = (b.x - a.z) * (pv - a.w) - (b.y - a.w) * (pu - a.z);
    const float e2 = (a.x - b.x) * (pv - b.y) - (a.y - b.y) * (pu - b.x);
    r.iA = 1.0f / (e0 + e1 + e2);
    r.lam[0] = e1 * r.iA; r.lam[1] = e2 * r.iA; r.lam[2] = e0 * r.iA;
    const float u0 = fminf(fmaxf(r.lam[0], 0.f), 1.f), u1 = fminf(fmaxf(r.lam[1], 0.f), 1.f), u2 = fminf(fmaxf(r.lam[2], 0.f), 1.f);
    r.isu = 1.0f / (u0 + u1 + u2);
    r.w[0] = u0 * r.isu; r.w[1] = u1 * r.isu; r.w[2] = u2 * r.isu;
    const float z = r.w[0] * c[0].x + r.w[1] * c[1].x + r.w[2] * c[2].x;
    r.e = (sh.far_z - z) * sh.inv_range * sh.inv_gamma;
    r.C[0] = r.w[0] * c[0].y + r.w[1] * c[1].y + r.w[2] * c[2].y;
    r.C[1] = r.w[0] * c[0].z + r.w[1] * c[1].z + r.w[2] * c[2].z;
    r.C[2] = r.w[0] * c[0].w + r.w[1] * c[1].w + r.w[2] * c[2].w;
}
// running softmax sums of one pixel: m = largest exponent so far, den / num relative to it
struct RgbAcc {
    float m, den, num[3];
    __device__ __forceinline__ RgbAcc(const ShadeDev &sh) : m(sh.eps_g), den(1.0f) { num[0] = sh.bg[0]; num[1] = sh.bg[1]; num[2] = sh.bg[2]; }
    __device__ __forceinline__ void add(const RgbTerm &r) {
        if (r.e > m) {
            const float f = expf(m - r.e);
            den *= f; num[0] *= f; num[1] *= f; num[2] *= f;
            m = r.e;
        }
        const float a = r.D * expf(r.e - m);
        den += a; num[0] += a * r.C[0]; num[1] += a * r.C[1]; num[2] += a * r.C[2];
    }
};

// grid (tiles_x, tiles_y, E).  image [E][3][H][W] out (may be null); target likewise / loss [E] (atomicAdd) optional.
__global__ void __launch_bounds__(kRsTile *kRsTile) k_rs_forward_rgb(CamDev cam, ShadeDev sh, int Mt, const TriRec *__restrict__ rec, const TriCol *__restrict__ col,
                                                                      float *__restrict__ image, const float *__restrict__ target, float scale,
                                                                      float *__restrict__ loss) {
    __shared__ float4 sa[kRsChunk], sb[kRsChunk], sc[3 * kRsChunk];
    __shared__ int sj[kRsChunk], s_cnt;
    __shared__ float red[8];
    const int env = blockIdx.z, pi = blockIdx.x * kRsTile + threadIdx.x, pj = blockIdx.y * kRsTile + threadIdx.y;
    const float su = 2.0f / cam.W, sv = 2.0f / cam.H;
    const float pu = (pi + 0.5f) * su - 1.0f, pv = (pj + 0.5f) * sv - 1.0f;
    const float tu0 = blockIdx.x * kRsTile * su - 1.0f, tv0 = blockIdx.y * kRsTile * sv - 1.0f, tu1 = tu0 + kRsTile * su, tv1 = tv0 + kRsTile * sv;
    RgbAcc acc(sh);
    for (int j0 = 0; j0 < Mt; j0 += kRsChunk) {
        const int n = stage_tris_rgb(rec + (size_t)env * Mt, col + (size_t)env * Mt, j0, Mt, tu0, tv0, tu1, tv1, sa, sb, sc, sj, &s_cnt);
        for (int q = 0; q < n; q++) {
            RgbTerm r;
            rgb_term(cam, sh, pu, pv, sa[q], sb[q], sc + 3 * q, r);
            if (r.on) acc.add(r);
        }
        __syncthreads();
    }
    const bool in = pi < cam.W && pj < cam.H;
    const size_t plane = (size_t)cam.H * cam.W, o = (size_t)env * 3 * plane + (size_t)pj * cam.W + pi;
    const float iden = 1.0f / acc.den;
    float d = 0.f;
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const float I = acc.num[c] * iden;
        if (in && image) image[o + c * plane] = I;
        if (in && target) { const float dd = I - target[o + c * plane]; d += dd * dd; }
    }
    if (target) {
        for (int w = 16; w > 0; w >>= 1) d += __shfl_xor_sync(0xffffffffu, d, w);
        const int tid = threadIdx.y * kRsTile + threadIdx.x;
        if ((tid & 31) == 0) red[tid >> 5] = d;
        __syncthreads();
        if (tid == 0) {
            float tot = 0.f;
            for (int w = 0; w < 8; w++) tot += red[w];
            atomicAdd(loss + env, scale * tot);
        }
    }
}

// Transposing warp sum: every lane brings K <= 32 values g[0..K) (the rest of the 32 slots count as zero); afterwards lane L
// holds the warp's total of component L.  Halving exchanges (16 + 8 + 4 + 2 + 1 = 31 shuffles instead of 5 K).
template <int K>
__device__ __forceinline__ float warp_transpose_sum(const float *g, int lane) {
    float h[16], q[8], r4[4], r2[2];
    const bool b4 = lane & 16, b3 = lane & 8, b2 = lane & 4, b1 = lane & 2, b0 = lane & 1;
#pragma unroll
    for (int i = 0; i < 16; i++) {
        const float lo = i < K ? g[i] : 0.f, hi = 16 + i < K ? g[16 + i] : 0.f;
        h[i] = (b4 ? hi : lo) + __shfl_xor_sync(0xffffffffu, b4 ? lo : hi, 16);
    }
#pragma unroll
    for (int i = 0; i < 8; i++) q[i] = (b3 ? h[8 + i] : h[i]) + __shfl_xor_sync(0xffffffffu, b3 ? h[i] : h[8 + i], 8);
#pragma unroll
    for (int i = 0; i < 4; i++) r4[i] = (b2 ? q[4 + i] : q[i]) + __shfl_xor_sync(0xffffffffu, b2 ? q[i] : q[4 + i], 4);
#pragma unroll
    for (int i = 0; i < 2; i++) r2[i] = (b1 ? r4[2 + i] : r4[i]) + __shfl_xor_sync(0xffffffffu, b1 ? r4[i] : r4[2 + i], 2);
    return (b0 ? r2[1] : r2[0]) + __shfl_xor_sync(0xffffffffu, b0 ? r2[0] : r2[1], 1);
}

// dL/d(NDC u, v and camera depth Z of the vertices) [E][N] float4 (x, y, z; zero on entry) and dL/dcolour [E][N][3] (zero on
// entry, may be null) of L = scale sum_{p, c} (I_c - I*_c)^2.  Pass 1 rebuilds the pixel's softmax sums; pass 2, per surviving
// triangle:  a = D e^{e - m},  g_a = sum_c gI_c (C_c - I_c) / W,  gC_c = gI_c a / W;  through the coverage ds as in the
// silhouette with dL/ds = g_a a (1 - D) / sigma;  through depth g_z = -g_a a / (gamma (far - near));  g_w_k = g_z Z_k +
// sum_c gC_c c_kc;  through w = u / sum u, u = clip(lam): g_lam_k = (g_w_k - sum_i g_w_i w_i) / sum u where 0 < lam_k < 1;
// through lam = (e_1, e_2, e_0) / (e_0 + e_1 + e_2) and the edge functions to the vertices.  The 18 per-vertex components
// are summed over the warp by shuffles; lane 0 issues the atomics.
__global__ void __launch_bounds__(kRsTile *kRsTile) k_rs_backward_rgb(CamDev cam, ShadeDev sh, int N, int Mt, const int *__restrict__ tris,
                                                                       const TriRec *__restrict__ rec, const TriCol *__restrict__ col,
                                                                       const float *__restrict__ target, float scale, float4 *__restrict__ g_ndc,
                                                                       float *__restrict__ g_colour) {
    __shared__ float4 sa[kRsChunk], sb[kRsChunk], sc[3 * kRsChunk];
    __shared__ int sj[kRsChunk], s_cnt;
    const int env = blockIdx.z, pi = blockIdx.x * kRsTile + threadIdx.x, pj = blockIdx.y * kRsTile + threadIdx.y;
    const float su = 2.0f / cam.W, sv = 2.0f / cam.H;
    const float pu = (pi + 0.5f) * su - 1.0f, pv = (pj + 0.5f) * sv - 1.0f;
    const float tu0 = blockIdx.x * kRsTile * su - 1.0f, tv0 = blockIdx.y * kRsTile * sv - 1.0f, tu1 = tu0 + kRsTile * su, tv1 = tv0 + kRsTile * sv;
    const TriRec *re = rec + (size_t)env * Mt;
    const TriCol *ce = col + (size_t)env * Mt;
    const bool in = pi < cam.W && pj < cam.H;
    const int lane = (threadIdx.y * kRsTile + threadIdx.x) & 31;
    RgbAcc acc(sh);
    for (int j0 = 0; j0 < Mt; j0 += kRsChunk) {
        const int n = stage_tris_rgb(re, ce, j0, Mt, tu0, tv0, tu1, tv1, sa, sb, sc, sj, &s_cnt);
        for (int q = 0; q < n; q++) {
            RgbTerm r;
            rgb_term(cam, sh, pu, pv, sa[q], sb[q], sc + 3 * q, r);
            if (r.on) acc.add(r);
        }
        __syncthreads();
    }
    const size_t plane = (size_t)cam.H * cam.W, o = (size_t)env * 3 * plane + (size_t)pj * cam.W + pi;
    const float iW = 1.0f / acc.den;
    float I[3], gI[3];
#pragma unroll
    for (int c = 0; c < 3; c++) {
        I[c] = acc.num[c] * iW;
        gI[c] = in ? 2.0f * scale * (I[c] - target[o + c * plane]) : 0.f;
    }
    const bool live = gI[0] != 0.f || gI[1] != 0.f || gI[2] != 0.f;
    for (int j0 = 0; j0 < Mt; j0 += kRsChunk) {
        const int n = stage_tris_rgb(re, ce, j0, Mt, tu0, tv0, tu1, tv1, sa, sb, sc, sj, &s_cnt);
        for (int q = 0; q < n; q++) {
            RgbTerm r;
            const float4 a4 = sa[q], b4 = sb[q];
            const float4 *cq = sc + 3 * q;
            rgb_term(cam, sh, pu, pv, a4, b4, cq, r);
            const bool use = live && r.on;
            if (!__any_sync(0xffffffffu, use)) continue;
            float g[18];  // NDC (u, v) of vertices 0, 1, 2; Z of 0, 1, 2; colour (r, g, b) of 0, 1, 2
#pragma unroll
            for (int i = 0; i < 18; i++) g[i] = 0.f;
            if (use) {
                const float a = r.D * expf(r.e - acc.m);
                const float g_a = (gI[0] * (r.C[0] - I[0]) + gI[1] * (r.C[1] - I[1]) + gI[2] * (r.C[2] - I[2])) * iW;
                const float gC[3] = {gI[0] * a * iW, gI[1] * a * iW, gI[2] * a * iW};
                // coverage: closest edge r.k -> r.k + 1
                const float gs = g_a * a * r.omD * cam.inv_sigma * (r.s >= 0.f ? 1.0f : -1.0f);
                const float wa = -2.0f * (1.0f - r.t) * gs, wb = -2.0f * r.t * gs;
                const int ka = r.k, kb = r.k == 2 ? 0 : r.k + 1;
#pragma unroll
                for (int v = 0; v < 3; v++) {
                    const float w = (v == ka ? wa : 0.f) + (v == kb ? wb : 0.f);
                    g[2 * v] = w * r.du; g[2 * v + 1] = w * r.dv;
                }
                // depth and colour through the clamped barycentrics
                const float g_z = -(g_a * a * sh.inv_gamma) * sh.inv_range;
                float g_w[3], dot = 0.f;
#pragma unroll
                for (int v = 0; v < 3; v++) {
                    g_w[v] = g_z * cq[v].x + gC[0] * cq[v].y + gC[1] * cq[v].z + gC[2] * cq[v].w;
                    dot += g_w[v] * r.w[v];
                    g[6 + v] = g_z * r.w[v];
                    g[9 + 3 * v] = gC[0] * r.w[v]; g[10 + 3 * v] = gC[1] * r.w[v]; g[11 + 3 * v] = gC[2] * r.w[v];
                }
                float g_lam[3], g_A2 = 0.f;
#pragma unroll
                for (int v = 0; v < 3; v++) {
                    g_lam[v] = (r.lam[v] > 0.f && r.lam[v] < 1.f) ? (g_w[v] - dot) * r.isu : 0.f;
                    g_A2 -= g_lam[v] * r.lam[v];
                }
                g_A2 *= r.iA;
                const float g_e[3] = {g_lam[2] * r.iA + g_A2, g_lam[0] * r.iA + g_A2, g_lam[1] * r.iA + g_A2};
                const float qu[3] = {a4.x, a4.z, b4.x}, qv[3] = {a4.y, a4.w, b4.y};
#pragma unroll
                for (int v = 0; v < 3; v++) {  // e_v = (qb_u - qa_u)(p_v - qa_v) - (qb_v - qa_v)(p_u - qa_u), qa = q_v, qb = q_{v+1}
                    const int vb = v == 2 ? 0 : v + 1;
                    g[2 * v] += g_e[v] * (qv[vb] - pv); g[2 * v + 1] += g_e[v] * (pu - qu[vb]);
                    g[2 * vb] += g_e[v] * (pv - qv[v]); g[2 * vb + 1] -= g_e[v] * (pu - qu[v]);
                }
            }
            // lane L ends up with the warp's total of component L (0-5 NDC, 6-8 depth, 9-17 colour) and issues its own atomic
            const float tot = warp_transpose_sum<18>(g, lane);
            if (lane < 18 && tot != 0.f) {
                const int *tr = tris + 3 * (size_t)sj[q];
                if (lane < 6) {
                    float4 *gn = g_ndc + (size_t)env * N + tr[lane >> 1];
                    atomicAdd((lane & 1) ? &gn->y : &gn->x, tot);
                } else if (lane < 9) {
                    atomicAdd(&g_ndc[(size_t)env * N + tr[lane - 6]].z, tot);
                } else if (g_colour) {
                    const int v = (lane - 9) / 3, c = (lane - 9) - 3 * v;
                    atomicAdd(g_colour + 3 * ((size_t)env * N + tr[v]) + c, tot);
                }
            }
        }
        __syncthreads();
    }
}

// as k_rs_project_adj with the cotangent of the camera depth added: g = (dL/du, dL/dv, dL/dZ, -)
__global__ void k_rs_project_adj_rgb(CamDev cam, int E, int N, const float *__restrict__ x, const float4 *__restrict__ g_ndc, float *__restrict__ adj_x) {
    const size_t total = (size_t)E * N;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        const float px = x[3 * i], py = x[3 * i + 1], pz = x[3 * i + 2];
        const float X = cam.R[0] * px + cam.R[1] * py + cam.R[2] * pz + cam.t[0];
        const float Y = cam.R[3] * px + cam.R[4] * py + cam.R[5] * pz + cam.t[1];
        const float Z = cam.R[6] * px + cam.R[7] * py + cam.R[8] * pz + cam.t[2];
        float gx = 0.f, gy = 0.f, gz = 0.f;
        if (Z > cam.near_z) {
            const float4 g = g_ndc[i];
            const float iz = 1.0f / Z;
            gx = g.x * cam.fx * iz; gy = g.y * cam.fy * iz; gz = -(g.x * cam.fx * X + g.y * cam.fy * Y) * iz * iz + g.z;
        }
        adj_x[3 * i] = cam.R[0] * gx + cam.R[3] * gy + cam.R[6] * gz;
        adj_x[3 * i + 1] = cam.R[1] * gx + cam.R[4] * gy + cam.R[7] * gz;
        adj_x[3 * i + 2] = cam.R[2] * gx + cam.R[5] * gy + cam.R[8] * gz;
    }
}

static int grid1(size_t n) { size_t g = (n + 255) / 256; return (int)(g < 1 ? 1 : (g > 148 * 16 ? 148 * 16 : g)); }
static size_t al256r(size_t n) { return (n + 255) & ~(size_t)255; }

}  // namespace gs

using namespace gs;

static int cam_dev(const gs_camera *c, CamDev *d) {
    if (!c) { set_error("camera is null"); return GS_EINVAL; }
    if (c->width < 1 || c->height < 1 || !(c->sigma > 0.f) || !(c->fx != 0.f) || !(c->fy != 0.f)) { set_error("bad camera: width, height >= 1, sigma > 0, fx, fy != 0"); return GS_EINVAL; }
    for (int i = 0; i < 9; i++) d->R[i] = c->R[i];
    for (int i = 0; i < 3; i++) d->t[i] = c->t[i];
    d->fx = c->fx; d->fy = c->fy; d->sigma = c->sigma; d->near_z = c->near_z; d->inv_sigma = 1.0f / c->sigma;
    d->cull_r = sqrtf(kRsCull * c->sigma);
    d->W = c->width; d->H = c->height;
    return GS_OK;
}

extern "C" size_t gs_raster_scratch_bytes(int n_envs, int n_particles, int n_tris) {
    if (n_envs < 1 || n_particles < 1 || n_tris < 0) return 0;
    return al256r((size_t)n_envs * n_particles * sizeof(float4)) + al256r((size_t)n_envs * n_particles * sizeof(float2)) +
           al256r((size_t)n_envs * (n_tris ? n_tris : 1) * sizeof(TriRec)) + 256;
}

static int raster_run(int E, int N, const float *d_x, int Mt, const int32_t *d_tris, const gs_camera *cam, float *d_image, const float *d_target, float scale,
                      int accumulate, float *d_loss, float *d_adj_x, void *d_scratch, size_t bytes, cudaStream_t st) {
    CamDev cd;
    int rc = cam_dev(cam, &cd);
    if (rc != GS_OK) return rc;
    if (E < 1 || N < 1 || Mt < 0 || !d_x || (Mt > 0 && !d_tris) || !d_scratch) { set_error("bad argument"); return GS_EINVAL; }
    if (bytes < gs_raster_scratch_bytes(E, N, Mt) || ((uintptr_t)d_scratch & 255)) { set_error("raster scratch too small or misaligned"); return GS_EINVAL; }
    if (E > 65535) { set_error("at most 65535 environments per render call"); return GS_EINVAL; }
    char *p = (char *)d_scratch;
    float4 *ndc = (float4 *)p; p += al256r((size_t)E * N * sizeof(float4));
    float2 *g_ndc = (float2 *)p; p += al256r((size_t)E * N * sizeof(float2));
    TriRec *rec = (TriRec *)p;
    const dim3 grid((cd.W + kRsTile - 1) / kRsTile, (cd.H + kRsTile - 1) / kRsTile, E), block(kRsTile, kRsTile);
    k_rs_project<<<grid1((size_t)E * N), 256, 0, st>>>(cd, E, N, d_x, ndc);
    if (Mt > 0) k_rs_pack<<<grid1((size_t)E * Mt), 256, 0, st>>>(cd, E, N, Mt, d_tris, ndc, rec);
    count_launch(Mt > 0 ? 2 : 1);
    if (d_loss && !accumulate) { cudaError_t e = cudaMemsetAsync(d_loss, 0, sizeof(float) * E, st); if (e != cudaSuccess) return cuda_fail(e, "zero loss"); }
    k_rs_forward<<<grid, block, 0, st>>>(cd, Mt, rec, d_image, d_target, scale, d_loss);
    count_launch();
    if (d_adj_x) {
        cudaError_t e = cudaMemsetAsync(g_ndc, 0, sizeof(float2) * (size_t)E * N, st);
        if (e != cudaSuccess) return cuda_fail(e, "zero NDC gradients");
        if (Mt > 0) { k_rs_backward<<<grid, block, 0, st>>>(cd, N, Mt, d_tris, rec, d_target, scale, g_ndc); count_launch(); }
        k_rs_project_adj<<<grid1((size_t)E * N), 256, 0, st>>>(cd, E, N, d_x, g_ndc, d_adj_x);
        count_launch();
    }
    cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? GS_OK : cuda_fail(e, "raster kernels");
}

extern "C" int gs_render_silhouette(int n_envs, int n_particles, const float *d_x, int n_tris, const int32_t *d_tris, const gs_camera *cam, float *d_image,
                                    void *d_scratch, size_t scratch_bytes, gs_stream stream) {
    if (!d_image) { set_error("image is null"); return GS_EINVAL; }
    return raster_run(n_envs, n_particles, d_x, n_tris, d_tris, cam, d_image, nullptr, 0.f, 0, nullptr, nullptr, d_scratch, scratch_bytes, (cudaStream_t)stream);
}

extern "C" int gs_loss_silhouette(int n_envs, int n_particles, const float *d_x, int n_tris, const int32_t *d_tris, const gs_camera *cam, const float *d_target,
                                  float scale, int accumulate, float *d_loss, float *d_adj_x, float *d_image, void *d_scratch, size_t scratch_bytes,
                                  gs_stream stream) {
    if (!d_target || !d_loss) { set_error("target and loss are required"); return GS_EINVAL; }
    return raster_run(n_envs, n_particles, d_x, n_tris, d_tris, cam, d_image, d_target, scale, accumulate, d_loss, d_adj_x, d_scratch, scratch_bytes,
                      (cudaStream_t)stream);
}

// ------------------------------------------------------------------------------------------ colour channel: entry points
static int shade_dev(const gs_shading *s, const gs_camera *c, ShadeDev *d) {
    if (!s) { set_error("shading is null"); return GS_EINVAL; }
    if (!(s->gamma > 0.f) || !(s->far_z > c->near_z)) { set_error("bad shading: gamma > 0, far_z > near_z"); return GS_EINVAL; }
    d->inv_gamma = 1.0f / s->gamma;
    d->eps_g = s->eps / s->gamma;
    d->far_z = s->far_z;
    d->inv_range = 1.0f / (s->far_z - c->near_z);
    for (int i = 0; i < 3; i++) d->bg[i] = s->background[i];
    d->s_cut = -kRsCull * c->sigma;
    return GS_OK;
}

extern "C" size_t gs_raster_rgb_scratch_bytes(int n_envs, int n_particles, int n_tris) {
    if (n_envs < 1 || n_particles < 1 || n_tris < 0) return 0;
    const size_t mt = n_tris ? n_tris : 1;
    return 2 * al256r((size_t)n_envs * n_particles * sizeof(float4)) + al256r((size_t)n_envs * mt * sizeof(TriRec)) +
           al256r((size_t)n_envs * mt * sizeof(TriCol)) + 256;
}

static int raster_run_rgb(int E, int N, const float *d_x, int Mt, const int32_t *d_tris, const float *d_colour, const gs_camera *cam, const gs_shading *shading,
                          float *d_image, const float *d_target, float scale, int accumulate, float *d_loss, float *d_adj_x, float *d_adj_colour,
                          void *d_scratch, size_t bytes, cudaStream_t st) {
    CamDev cd;
    ShadeDev sd;
    int rc = cam_dev(cam, &cd);
    if (rc == GS_OK) rc = shade_dev(shading, cam, &sd);
    if (rc != GS_OK) return rc;
    if (E < 1 || N < 1 || Mt < 0 || !d_x || !d_colour || (Mt > 0 && !d_tris) || !d_scratch) { set_error("bad argument"); return GS_EINVAL; }
    if (bytes < gs_raster_rgb_scratch_bytes(E, N, Mt) || ((uintptr_t)d_scratch & 255)) { set_error("raster scratch too small or misaligned"); return GS_EINVAL; }
    if (E > 65535) { set_error("at most 65535 environments per render call"); return GS_EINVAL; }
    char *p = (char *)d_scratch;
    float4 *ndc = (float4 *)p; p += al256r((size_t)E * N * sizeof(float4));
    float4 *g_ndc = (float4 *)p; p += al256r((size_t)E * N * sizeof(float4));
    TriRec *rec = (TriRec *)p; p += al256r((size_t)E * (Mt ? Mt : 1) * sizeof(TriRec));
    TriCol *col = (TriCol *)p;
    const dim3 grid((cd.W + kRsTile - 1) / kRsTile, (cd.H + kRsTile - 1) / kRsTile, E), block(kRsTile, kRsTile);
    k_rs_project<<<grid1((size_t)E * N), 256, 0, st>>>(cd, E, N, d_x, ndc);
    count_launch();
    if (Mt > 0) {
        k_rs_pack<<<grid1((size_t)E * Mt), 256, 0, st>>>(cd, E, N, Mt, d_tris, ndc, rec);
        k_rs_pack_rgb<<<grid1((size_t)E * Mt), 256, 0, st>>>(E, N, Mt, d_tris, ndc, d_colour, rec, col);
        count_launch(2);
    }
    cudaError_t e = cudaSuccess;
    if (d_loss && !accumulate) e = cudaMemsetAsync(d_loss, 0, sizeof(float) * E, st);
    if (e != cudaSuccess) return cuda_fail(e, "zero loss");
    k_rs_forward_rgb<<<grid, block, 0, st>>>(cd, sd, Mt, rec, col, d_image, d_target, scale, d_loss);
    count_launch();
    if (d_adj_x || d_adj_colour) {
        e = cudaMemsetAsync(g_ndc, 0, sizeof(float4) * (size_t)E * N, st);
        if (e == cudaSuccess && d_adj_colour) e = cudaMemsetAsync(d_adj_colour, 0, sizeof(float) * 3 * (size_t)E * N, st);
        if (e != cudaSuccess) return cuda_fail(e, "zero raster gradients");
        if (Mt > 0) { k_rs_backward_rgb<<<grid, block, 0, st>>>(cd, sd, N, Mt, d_tris, rec, col, d_target, scale, g_ndc, d_adj_colour); count_launch(); }
        if (d_adj_x) { k_rs_project_adj_rgb<<<grid1((size_t)E * N), 256, 0, st>>>(cd, E, N, d_x, g_ndc, d_adj_x); count_launch(); }
    }
    e = cudaGetLastError();
    return e == cudaSuccess ? GS_OK : cuda_fail(e, "raster kernels");
}

extern "C" int gs_render_rgb(int n_envs, int n_particles, const float *d_x, int n_tris, const int32_t *d_tris, const float *d_colour, const gs_camera *cam,
                             const gs_shading *shading, float *d_image, void *d_scratch, size_t scratch_bytes, gs_stream stream) {
    if (!d_image) { set_error("image is null"); return GS_EINVAL; }
    return raster_run_rgb(n_envs, n_particles, d_x, n_tris, d_tris, d_colour, cam, shading, d_image, nullptr, 0.f, 0, nullptr, nullptr, nullptr, d_scratch,
                          scratch_bytes, (cudaStream_t)stream);
}

extern "C" int gs_loss_rgb(int n_envs, int n_particles, const float *d_x, int n_tris, const int32_t *d_tris, const float *d_colour, const gs_camera *cam,
                           const gs_shading *shading, const float *d_target, float scale, int accumulate, float *d_loss, float *d_adj_x,
                           float *d_adj_colour, float *d_image, void *d_scratch, size_t scratch_bytes, gs_stream stream) {
    if (!d_target || !d_loss) { set_error("target and loss are required"); return GS_EINVAL; }
    return raster_run_rgb(n_envs, n_particles, d_x, n_tris, d_tris, d_colour, cam, shading, d_image, d_target, scale, accumulate, d_loss, d_adj_x,
                          d_adj_colour, d_scratch, scratch_bytes, (cudaStream_t)stream);
}

// ------------------------------------------------------------------------------------------ entry point that allocates nothing
// gs_loss_silhouette_static: gs_loss_silhouette with the scratch block (NDC vertices, NDC gradients, triangle records) in a
// file-scope device array instead of a caller block, for callers that cannot allocate (CUDA graph capture, serving loops).
// GS_RASTER_STATIC_BYTES of every GPU that loads the library are held until the process exits.  In host code the array's
// name is a host-side stand-in, not a device address: the address is taken with cudaGetSymbolAddress, once per device, with
// that device current, and passed to the kernels like any other scratch pointer.
static __device__ __align__(256) unsigned char g_rs_static[GS_RASTER_STATIC_BYTES];

#include <mutex>
static int raster_static_ptr(void **out) {
    constexpr int kMaxDev = 64;
    static std::mutex mu;
    static void *ptrs[kMaxDev] = {};
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e, "cudaGetDevice (static raster scratch)");
    if (dev < 0 || dev >= kMaxDev) { set_error("static raster scratch: device ordinal %d out of range", dev); return GS_EINVAL; }
    std::lock_guard<std::mutex> lock(mu);
    if (!ptrs[dev]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_rs_static);  // of the CURRENT device's copy of the array
        if (e != cudaSuccess || !p) return cuda_fail(e, "cudaGetSymbolAddress (static raster scratch)");
        ptrs[dev] = p;
    }
    *out = ptrs[dev];
    return GS_OK;
}

extern "C" int gs_loss_silhouette_static(int n_envs, int n_particles, const float *d_x, int n_tris, const int32_t *d_tris, const gs_camera *cam,
                                         const float *d_target, float scale, int accumulate, float *d_loss, float *d_adj_x, float *d_image,
                                         gs_stream stream) {
    if (!d_target || !d_loss) { set_error("target and loss are required"); return GS_EINVAL; }
    // sizes first: no CUDA call is made for a problem the block cannot hold
    const size_t need = gs_raster_scratch_bytes(n_envs, n_particles, n_tris);
    if (need == 0) { set_error("bad argument: n_envs, n_particles >= 1, n_tris >= 0"); return GS_EINVAL; }
    if (need > (size_t)GS_RASTER_STATIC_BYTES) {
        set_error("gs_loss_silhouette_static: this problem needs %zu bytes of scratch, the static block holds %zu (GS_RASTER_STATIC_BYTES); "
                  "use gs_loss_silhouette with a caller block",
                  need, (size_t)GS_RASTER_STATIC_BYTES);
        return GS_EINVAL;
    }
    void *scratch = nullptr;
    const int rc = raster_static_ptr(&scratch);
    if (rc != GS_OK) return rc;
    // the block keeps the previous call's contents: the NDC vertices and the triangle records are fully rewritten by
    // k_rs_project / k_rs_pack for this call's sizes, the NDC gradients and (unless accumulate) the loss are zeroed by
    // raster_run (cudaMemsetAsync on the stream: no allocation) before the adjoint adds into them
    return raster_run(n_envs, n_particles, d_x, n_tris, d_tris, cam, d_image, d_target, scale, accumulate, d_loss, d_adj_x, scratch,
                      (size_t)GS_RASTER_STATIC_BYTES, (cudaStream_t)stream);
}
