// gs_raster.cu -- soft silhouette rasteriser on a headless device buffer and its adjoint.
//
// PAPER.md:168-172 (section 2.2): the renderers "replace discontinuous triangle mesh edges with smooth sigmoids ... blurring
// triangle edges into semi-transparent boundaries".  The paper prints no formula; reading A22 takes the SoftRas
// silhouette as SPEC.md:251 states it:
//     D_j(p) = sigmoid(delta_j(p) d^2(p, boundary of triangle j) / sigma),  delta = +1 inside, -1 outside (NDC distances)
//     S(p)   = 1 - prod_j (1 - D_j(p));     loss ("pixelwise MSE")  L = scale sum_p (S(p) - S*(p))^2
// Camera: pinhole, p_cam = R x + t, drawn iff z_cam > near for all three vertices, NDC (u, v) = (fx X / Z, fy Y / Z), pixel
// (i, j) centre at u = 2 (i + 1/2) / W - 1, v = 2 (j + 1/2) / H - 1.  Silhouette channel only (no colour / texture shading).
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
