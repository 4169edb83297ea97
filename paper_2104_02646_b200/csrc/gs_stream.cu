// gs_stream.cu -- the STREAMING plan: two grid-wide kernels per substep.
//
//   k_elements_fwd   one CTA per tile of kTileElems Morton-ordered elements (tets, triangles and hinges in ONE
//                    launch, CTA ranges per type).  The tile's particles are staged in shared memory (float4
//                    gathers through a tile-local particle list), each thread evaluates one element with 16-bit
//                    local indices, writes its per-vertex forces to conflict-free shared-memory slots, and a
//                    per-tile-particle gather list sums them (no shared-memory atomics: fp32 smem atomics are CAS
//                    loops on sm_100a).  One REDG.E.ADD.F32x4 per tile-particle goes to the global force array.
//   k_particles_fwd  per particle: contact + friction from (x-, v-), semi-implicit Euler, writes the next tape
//                    slot, re-zeroes the force accumulator, flags non-finite states.
//   k_particles_adj  adjoint of integrate + contact; mass gradient; produces adj_f.
//   k_elements_adj   gather-form VJP of the element forces with the same tiles; parameter gradients.
//
// a1-a10 of SURVEY.md 8(a); citations of the formulas are in gs_elements.cuh.
#include <climits>

#include "gs_elements.cuh"
#include "gs_internal.h"

namespace gs {

#define GS_LAUNCH_CHECK(what)                                        \
    do {                                                             \
        cudaError_t e_ = cudaGetLastError();                         \
        if (e_ != cudaSuccess) return cuda_fail(e_, what);           \
        g_launches++;                                                \
    } while (0)
// GS_TIMED(m, id, st, what, launch): the launch, bracketed by events when the model's kernel timing is on
#define GS_TIMED(m, id, st, what, ...)                                 \
    do {                                                               \
        cudaEvent_t ta_ = (m)->timing ? timing_begin(m, st) : nullptr; \
        __VA_ARGS__;                                                   \
        GS_LAUNCH_CHECK(what);                                         \
        if (ta_) timing_end(m, id, ta_, st);                           \
    } while (0)

__device__ __forceinline__ void red_add_v4(float4 *addr, float a, float b, float c) {
    // one vector reduction per particle instead of three scalar ones (REDG.E.ADD.F32x4)
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(addr), "f"(a), "f"(b), "f"(c), "f"(0.0f) : "memory");
}

__device__ __forceinline__ int tile_type(const ModelDev &md, int tile) { return tile >= md.tile_begin[2] ? 2 : (tile >= md.tile_begin[1] ? 1 : 0); }

// ------------------------------------------------------------------------------------------ forward elements
__global__ void __launch_bounds__(kTileElems) k_elements_fwd(const ModelDev md, const float4 *__restrict__ x4, const float4 *__restrict__ v4,
                                                             float4 *__restrict__ f4, int pmax) {
    extern __shared__ float4 smem4[];
    float4 *sx = smem4, *sv = smem4 + pmax;
    float *sf = reinterpret_cast<float *>(smem4 + 2 * pmax);  // [3][4 * kTileElems]
    constexpr int PL = 4 * kTileElems;
    const int tid = threadIdx.x, env = blockIdx.y;
    const int type = tile_type(md, blockIdx.x);
    const ElemDev &es = md.es[type];
    const int j = blockIdx.x - md.tile_begin[type];
    const int p0 = es.tile_part_ptr[j], np = es.tile_part_ptr[j + 1] - p0;
    const size_t eoff = (size_t)env * md.N;
    for (int p = tid; p < np; p += kTileElems) {
        const int id = es.tile_parts[p0 + p];
        sx[p] = x4[eoff + id];
        if (type != T_HINGE) sv[p] = v4[eoff + id];
    }
    __syncthreads();
    const int e = j * kTileElems + tid;
    if (e < es.count) {
        const ushort4 li = es.lidx[e];
        if (type == T_TET) {
            const float4 c0 = es.c0[e], c1 = es.c1[e];
            const float2 c2 = es.c2[e];
            const float b[9] = {c0.x, c0.y, c0.z, c0.w, c1.x, c1.y, c1.z, c1.w, c2.x};
            const size_t pe = (size_t)env * es.count + e;
            const vec3 x[4] = {vec3(sx[li.x]), vec3(sx[li.y]), vec3(sx[li.z]), vec3(sx[li.w])};
            const vec3 v[4] = {vec3(sv[li.x]), vec3(sv[li.y]), vec3(sv[li.z]), vec3(sv[li.w])};
            vec3 f[4];
            tet_force(x, v, b, c2.y, es.mu[pe], es.lam[pe], es.damp[pe], f);
#pragma unroll
            for (int k = 0; k < 4; k++) { sf[k * kTileElems + tid] = f[k].x; sf[PL + k * kTileElems + tid] = f[k].y; sf[2 * PL + k * kTileElems + tid] = f[k].z; }
        } else if (type == T_TRI) {
            const float4 c0 = es.c0[e];
            const float A = es.c1[e].x;
            const float b[4] = {c0.x, c0.y, c0.z, c0.w};
            const size_t pe = (size_t)env * es.count + e;
            const vec3 x[3] = {vec3(sx[li.x]), vec3(sx[li.y]), vec3(sx[li.z])};
            const vec3 v[3] = {vec3(sv[li.x]), vec3(sv[li.y]), vec3(sv[li.z])};
            vec3 f[3];
            tri_force(x, v, b, A, es.mu[pe], es.lam[pe], es.damp[pe], f);
#pragma unroll
            for (int k = 0; k < 3; k++) { sf[k * kTileElems + tid] = f[k].x; sf[PL + k * kTileElems + tid] = f[k].y; sf[2 * PL + k * kTileElems + tid] = f[k].z; }
        } else {
            const float4 c0 = es.c0[e];
            const vec3 x[4] = {vec3(sx[li.x]), vec3(sx[li.y]), vec3(sx[li.z]), vec3(sx[li.w])};
            vec3 f[4];
            hinge_force(x, c0.x, c0.y, c0.z, f);
#pragma unroll
            for (int k = 0; k < 4; k++) { sf[k * kTileElems + tid] = f[k].x; sf[PL + k * kTileElems + tid] = f[k].y; sf[2 * PL + k * kTileElems + tid] = f[k].z; }
        }
    }
    __syncthreads();
    const int arity = type == T_TRI ? 3 : 4;
    const uint16_t *slots = es.csr_slots + (size_t)j * arity * kTileElems;
    for (int p = tid; p < np; p += kTileElems) {
        const int beg = p ? es.csr_end[p0 + p - 1] : 0, end = es.csr_end[p0 + p];
        float ax = 0.f, ay = 0.f, az = 0.f;
        for (int q = beg; q < end; q++) {
            const int s = slots[q];
            ax += sf[s]; ay += sf[PL + s]; az += sf[2 * PL + s];
        }
        red_add_v4(f4 + eoff + es.tile_parts[p0 + p], ax, ay, az);
    }
}

// ------------------------------------------------------------------------------------------ forward particles
__device__ __forceinline__ ContactParams contact_params(const ModelDev &md, int env) {
    ContactParams cp;
    cp.n = vec3(md.nx, md.ny, md.nz); cp.d = md.pd; cp.r = md.pr;
    cp.ke = md.ke[env]; cp.kd = md.kd[env]; cp.kf = md.kf[env]; cp.mu = md.muc[env];
    return cp;
}

__global__ void __launch_bounds__(256) k_particles_fwd(const ModelDev md, const float4 *__restrict__ x4, const float4 *__restrict__ v4,
                                                       float4 *__restrict__ f4, float4 *__restrict__ xo, float4 *__restrict__ vo, int substep) {
    const size_t total = (size_t)md.E * md.N;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        const int env = (int)(i / md.N);
        const float4 xq = x4[i], vq = v4[i], fq = f4[i];
        const ContactParams cp = contact_params(md, env);
        const vec3 x(xq), v(vq);
        const vec3 f = vec3(fq) + contact_force(cp, x, v);
        vec3 x1, v1;
        integrate(x, v, f, xq.w, vec3(md.gx, md.gy, md.gz), md.dt, x1, v1);
        xo[i] = make_float4(x1.x, x1.y, x1.z, xq.w);
        vo[i] = make_float4(v1.x, v1.y, v1.z, 0.f);
        f4[i] = make_float4(0.f, 0.f, 0.f, 0.f);
        const float chk = x1.x + x1.y + x1.z + v1.x + v1.y + v1.z;
        if (!(fabsf(chk) <= 3.0e38f)) atomicMin(md.bad, substep);
    }
}

// ------------------------------------------------------------------------------------------ adjoint particles
// frame_cot: caller-order [E][N][3] cotangent dL/dx of the state AFTER this substep, or nullptr.
__global__ void __launch_bounds__(256) k_particles_adj(const ModelDev md, const float4 *__restrict__ x4, const float4 *__restrict__ v4,
                                                       const float4 *__restrict__ v4n, const float *__restrict__ frame_cot,
                                                       float4 *__restrict__ adjx, float4 *__restrict__ adjv, float4 *__restrict__ adjf) {
    const size_t total = (size_t)md.E * md.N;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        const int env = (int)(i / md.N), id = (int)(i - (size_t)env * md.N);
        const float4 xq = x4[i], vq = v4[i], vn = v4n[i];
        vec3 bx(adjx[i]), bv(adjv[i]);
        if (frame_cot) {
            const float *c = frame_cot + ((size_t)env * md.N + md.perm_p[id]) * 3;
            bx += vec3(c[0], c[1], c[2]);
        }
        const float w = xq.w, dt = md.dt;
        const vec3 x(xq), v(vq);
        const vec3 lv = madd(bv, dt, bx);  // cotangent of v+
        const vec3 af = (dt * w) * lv;
        vec3 ax = bx, av = lv;
        if (w > 0.0f) {
            // f w dt = v+ - v- - g dt  =>  dL/dm = -w^2 dt f.lv = -w (v+ - v- - g dt).lv   (A11)
            const vec3 dvf = (vec3(vn) - v) - dt * vec3(md.gx, md.gy, md.gz);
            md.gmass32[i] += -w * dot(dvf, lv);
        }
        contact_adjoint(contact_params(md, env), x, v, af, ax, av);
        adjx[i] = make_float4(ax.x, ax.y, ax.z, 0.f);
        adjv[i] = make_float4(av.x, av.y, av.z, 0.f);
        adjf[i] = make_float4(af.x, af.y, af.z, 0.f);
    }
}

// ------------------------------------------------------------------------------------------ adjoint elements
__global__ void __launch_bounds__(kTileElems) k_elements_adj(const ModelDev md, const float4 *__restrict__ x4, const float4 *__restrict__ v4,
                                                             const float4 *__restrict__ adjf, float4 *__restrict__ adjx, float4 *__restrict__ adjv, int pmax) {
    extern __shared__ float4 smem4[];
    float4 *sx = smem4, *sv = smem4 + pmax, *sa = smem4 + 2 * pmax;
    float *sf = reinterpret_cast<float *>(smem4 + 3 * pmax);  // [6][4 * kTileElems]: ax xyz, av xyz
    constexpr int PL = 4 * kTileElems;
    const int tid = threadIdx.x, env = blockIdx.y;
    const int type = tile_type(md, blockIdx.x);
    const ElemDev &es = md.es[type];
    const int j = blockIdx.x - md.tile_begin[type];
    const int p0 = es.tile_part_ptr[j], np = es.tile_part_ptr[j + 1] - p0;
    const size_t eoff = (size_t)env * md.N;
    for (int p = tid; p < np; p += kTileElems) {
        const int id = es.tile_parts[p0 + p];
        sx[p] = x4[eoff + id];
        sa[p] = adjf[eoff + id];
        if (type != T_HINGE) sv[p] = v4[eoff + id];
    }
    __syncthreads();
    const int e = j * kTileElems + tid;
    if (e < es.count) {
        const ushort4 li = es.lidx[e];
        if (type == T_TET) {
            const float4 c0 = es.c0[e], c1 = es.c1[e];
            const float2 c2 = es.c2[e];
            const float b[9] = {c0.x, c0.y, c0.z, c0.w, c1.x, c1.y, c1.z, c1.w, c2.x};
            const size_t pe = (size_t)env * es.count + e;
            const vec3 x[4] = {vec3(sx[li.x]), vec3(sx[li.y]), vec3(sx[li.z]), vec3(sx[li.w])};
            const vec3 v[4] = {vec3(sv[li.x]), vec3(sv[li.y]), vec3(sv[li.z]), vec3(sv[li.w])};
            const vec3 a[4] = {vec3(sa[li.x]), vec3(sa[li.y]), vec3(sa[li.z]), vec3(sa[li.w])};
            vec3 ax[4], av[4];
            float gmu, glam, gk;
            tet_adjoint(x, v, a, b, c2.y, es.mu[pe], es.lam[pe], es.damp[pe], ax, av, gmu, glam, gk);
            const size_t gs_ = (size_t)md.E * es.count;
            es.g32[pe] += gmu; es.g32[gs_ + pe] += glam; es.g32[2 * gs_ + pe] += gk;
#pragma unroll
            for (int k = 0; k < 4; k++) {
                sf[k * kTileElems + tid] = ax[k].x; sf[PL + k * kTileElems + tid] = ax[k].y; sf[2 * PL + k * kTileElems + tid] = ax[k].z;
                sf[3 * PL + k * kTileElems + tid] = av[k].x; sf[4 * PL + k * kTileElems + tid] = av[k].y; sf[5 * PL + k * kTileElems + tid] = av[k].z;
            }
        } else if (type == T_TRI) {
            const float4 c0 = es.c0[e];
            const float A = es.c1[e].x;
            const float b[4] = {c0.x, c0.y, c0.z, c0.w};
            const size_t pe = (size_t)env * es.count + e;
            const vec3 x[3] = {vec3(sx[li.x]), vec3(sx[li.y]), vec3(sx[li.z])};
            const vec3 v[3] = {vec3(sv[li.x]), vec3(sv[li.y]), vec3(sv[li.z])};
            const vec3 a[3] = {vec3(sa[li.x]), vec3(sa[li.y]), vec3(sa[li.z])};
            vec3 ax[3], av[3];
            float gmu, glam, gk;
            tri_adjoint(x, v, a, b, A, es.mu[pe], es.lam[pe], es.damp[pe], ax, av, gmu, glam, gk);
            const size_t gs_ = (size_t)md.E * es.count;
            es.g32[pe] += gmu; es.g32[gs_ + pe] += glam; es.g32[2 * gs_ + pe] += gk;
#pragma unroll
            for (int k = 0; k < 3; k++) {
                sf[k * kTileElems + tid] = ax[k].x; sf[PL + k * kTileElems + tid] = ax[k].y; sf[2 * PL + k * kTileElems + tid] = ax[k].z;
                sf[3 * PL + k * kTileElems + tid] = av[k].x; sf[4 * PL + k * kTileElems + tid] = av[k].y; sf[5 * PL + k * kTileElems + tid] = av[k].z;
            }
        } else {
            const float4 c0 = es.c0[e];
            const vec3 x[4] = {vec3(sx[li.x]), vec3(sx[li.y]), vec3(sx[li.z]), vec3(sx[li.w])};
            const vec3 a[4] = {vec3(sa[li.x]), vec3(sa[li.y]), vec3(sa[li.z]), vec3(sa[li.w])};
            vec3 ax[4];
            hinge_adjoint(x, a, c0.x, c0.y, c0.z, ax);
#pragma unroll
            for (int k = 0; k < 4; k++) { sf[k * kTileElems + tid] = ax[k].x; sf[PL + k * kTileElems + tid] = ax[k].y; sf[2 * PL + k * kTileElems + tid] = ax[k].z; }
        }
    }
    __syncthreads();
    const int arity = type == T_TRI ? 3 : 4;
    const uint16_t *slots = es.csr_slots + (size_t)j * arity * kTileElems;
    for (int p = tid; p < np; p += kTileElems) {
        const int beg = p ? es.csr_end[p0 + p - 1] : 0, end = es.csr_end[p0 + p];
        float ax = 0.f, ay = 0.f, az = 0.f, bx = 0.f, by = 0.f, bz = 0.f;
        if (type != T_HINGE) {
            for (int q = beg; q < end; q++) {
                const int s = slots[q];
                ax += sf[s]; ay += sf[PL + s]; az += sf[2 * PL + s];
                bx += sf[3 * PL + s]; by += sf[4 * PL + s]; bz += sf[5 * PL + s];
            }
        } else {
            for (int q = beg; q < end; q++) {
                const int s = slots[q];
                ax += sf[s]; ay += sf[PL + s]; az += sf[2 * PL + s];
            }
        }
        const int id = es.tile_parts[p0 + p];
        red_add_v4(adjx + eoff + id, ax, ay, az);
        if (type != T_HINGE) red_add_v4(adjv + eoff + id, bx, by, bz);
    }
}

// ------------------------------------------------------------------------------------------ layout conversion
// caller [E][N][3] -> internal float4 (x.w = inverse mass when x_is_state)
__global__ void k_pack(const ModelDev md, const float *__restrict__ x, const float *__restrict__ v, float4 *__restrict__ x4, float4 *__restrict__ v4, int x_is_state) {
    const size_t total = (size_t)md.E * md.N;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        const int env = (int)(i / md.N), id = (int)(i - (size_t)env * md.N);
        const size_t c = ((size_t)env * md.N + md.perm_p[id]) * 3;
        if (x4) x4[i] = x ? make_float4(x[c], x[c + 1], x[c + 2], x_is_state ? md.inv_mass[i] : 0.f) : make_float4(0.f, 0.f, 0.f, 0.f);
        if (v4) v4[i] = v ? make_float4(v[c], v[c + 1], v[c + 2], 0.f) : make_float4(0.f, 0.f, 0.f, 0.f);
    }
}
__global__ void k_unpack(const ModelDev md, const float4 *__restrict__ x4, const float4 *__restrict__ v4, float *__restrict__ x, float *__restrict__ v) {
    const size_t total = (size_t)md.E * md.N;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        const int env = (int)(i / md.N), id = (int)(i - (size_t)env * md.N);
        const size_t c = ((size_t)env * md.N + md.perm_p[id]) * 3;
        if (x) { const float4 q = x4[i]; x[c] = q.x; x[c + 1] = q.y; x[c + 2] = q.z; }
        if (v) { const float4 q = v4[i]; v[c] = q.x; v[c + 1] = q.y; v[c + 2] = q.z; }
    }
}

// ------------------------------------------------------------------------------------------ gradients / parameters
__global__ void k_flush(float *__restrict__ g32, double *__restrict__ g64, size_t n) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        g64[i] += (double)g32[i];
        g32[i] = 0.f;
    }
}
__global__ void k_zero(float *__restrict__ g32, double *__restrict__ g64, size_t n) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) { g64[i] = 0.0; g32[i] = 0.f; }
}
// out[env][perm[e]] = g64[env][e]
__global__ void k_get_grads(const double *__restrict__ g64, const int *__restrict__ perm, float *__restrict__ out, int E, int count) {
    const size_t total = (size_t)E * count;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        const int env = (int)(i / count), e = (int)(i - (size_t)env * count);
        out[(size_t)env * count + perm[e]] = (float)g64[i];
    }
}
__global__ void k_set_params(float *__restrict__ dst, const int *__restrict__ perm, const float *__restrict__ src, int E, int count, int as_inv_mass) {
    const size_t total = (size_t)E * count;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        const int env = (int)(i / count), e = (int)(i - (size_t)env * count);
        const float val = src[(size_t)env * count + perm[e]];
        if (as_inv_mass) { if (dst[i] != 0.f) dst[i] = 1.0f / val; }  // pinned particles stay pinned
        else dst[i] = val;
    }
}

// ------------------------------------------------------------------------------------------ host launches
static inline int grid_for(size_t n, int block = 256) {
    size_t g = (n + block - 1) / block;
    const size_t cap = 148 * 16;  // grid-stride beyond this
    return (int)(g < 1 ? 1 : (g > cap ? cap : g));
}

int configure_stream_kernels(gs_model *m) {
    int pmax = 1;
    for (int t = 0; t < N_TYPES; t++) pmax = pmax > m->hes[t].max_tile_parts ? pmax : m->hes[t].max_tile_parts;
    m->fwd_smem = 2 * pmax * (int)sizeof(float4) + 3 * 4 * kTileElems * (int)sizeof(float);
    m->adj_smem = 3 * pmax * (int)sizeof(float4) + 6 * 4 * kTileElems * (int)sizeof(float);
    cudaError_t e = cudaFuncSetAttribute(k_elements_fwd, cudaFuncAttributeMaxDynamicSharedMemorySize, m->fwd_smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_elements_adj, cudaFuncAttributeMaxDynamicSharedMemorySize, m->adj_smem);
    if (e != cudaSuccess) return cuda_fail(e, "cudaFuncSetAttribute");
    return GS_OK;
}

static inline int pmax_of(const gs_model *m) {
    int pmax = 1;
    for (int t = 0; t < N_TYPES; t++) pmax = pmax > m->hes[t].max_tile_parts ? pmax : m->hes[t].max_tile_parts;
    return pmax;
}

int stream_step_forward(gs_model *m, const float4 *x, const float4 *v, float4 *xo, float4 *vo, int substep, cudaStream_t st) {
    const int tiles = m->dev.tile_begin[N_TYPES];
    if (tiles > 0) {
        GS_TIMED(m, GS_K_ELEMENTS_FWD, st, "k_elements_fwd", k_elements_fwd<<<dim3(tiles, m->E), kTileElems, m->fwd_smem, st>>>(m->dev, x, v, m->d_f, pmax_of(m)));
    }
    GS_TIMED(m, GS_K_PARTICLES_FWD, st, "k_particles_fwd", k_particles_fwd<<<grid_for((size_t)m->E * m->N), 256, 0, st>>>(m->dev, x, v, m->d_f, xo, vo, substep));
    return GS_OK;
}

// adjoint of the substep whose start state is (x, v) and whose end velocity is v_next; cotangents live in
// m->d_adjx / m->d_adjv (updated in place); frame_cot (caller order, may be null) is added to adj_x first.
int stream_step_adjoint(gs_model *m, const float4 *x, const float4 *v, const float4 *v_next, const float *frame_cot, cudaStream_t st) {
    GS_TIMED(m, GS_K_PARTICLES_ADJ, st, "k_particles_adj",
             k_particles_adj<<<grid_for((size_t)m->E * m->N), 256, 0, st>>>(m->dev, x, v, v_next, frame_cot, m->d_adjx, m->d_adjv, m->d_adjf));
    const int tiles = m->dev.tile_begin[N_TYPES];
    if (tiles > 0) {
        GS_TIMED(m, GS_K_ELEMENTS_ADJ, st, "k_elements_adj",
                 k_elements_adj<<<dim3(tiles, m->E), kTileElems, m->adj_smem, st>>>(m->dev, x, v, m->d_adjf, m->d_adjx, m->d_adjv, pmax_of(m)));
    }
    if (++m->steps_since_flush >= kFlushEvery) return launch_flush_grads(m, st);
    return GS_OK;
}

int launch_pack(gs_model *m, const float *x, const float *v, float4 *x4, float4 *v4, bool x_is_state, cudaStream_t st) {
    GS_TIMED(m, GS_K_OTHER, st, "k_pack", k_pack<<<grid_for((size_t)m->E * m->N), 256, 0, st>>>(m->dev, x, v, x4, v4, x_is_state ? 1 : 0));
    return GS_OK;
}
int launch_unpack(gs_model *m, const float4 *x4, const float4 *v4, float *x, float *v, cudaStream_t st) {
    if (!x && !v) return GS_OK;
    GS_TIMED(m, GS_K_OTHER, st, "k_unpack", k_unpack<<<grid_for((size_t)m->E * m->N), 256, 0, st>>>(m->dev, x4, v4, x, v));
    return GS_OK;
}

int launch_flush_grads(gs_model *m, cudaStream_t st) {
    m->steps_since_flush = 0;
    for (int t = 0; t < 2; t++) {
        const size_t n = 3 * (size_t)m->E * m->counts[t];
        if (!n) continue;
        GS_TIMED(m, GS_K_OTHER, st, "k_flush", k_flush<<<grid_for(n), 256, 0, st>>>(m->dev.es[t].g32, m->dev.es[t].g64, n));
    }
    GS_TIMED(m, GS_K_OTHER, st, "k_flush", k_flush<<<grid_for((size_t)m->E * m->N), 256, 0, st>>>(m->dev.gmass32, m->dev.gmass64, (size_t)m->E * m->N));
    return GS_OK;
}
int launch_zero_grads(gs_model *m, cudaStream_t st) {
    m->steps_since_flush = 0;
    for (int t = 0; t < 2; t++) {
        const size_t n = 3 * (size_t)m->E * m->counts[t];
        if (!n) continue;
        GS_TIMED(m, GS_K_OTHER, st, "k_zero", k_zero<<<grid_for(n), 256, 0, st>>>(m->dev.es[t].g32, m->dev.es[t].g64, n));
    }
    GS_TIMED(m, GS_K_OTHER, st, "k_zero", k_zero<<<grid_for((size_t)m->E * m->N), 256, 0, st>>>(m->dev.gmass32, m->dev.gmass64, (size_t)m->E * m->N));
    return GS_OK;
}
int launch_get_grads(gs_model *m, int group, float *d_out, cudaStream_t st) {
    int rc = launch_flush_grads(m, st);
    if (rc != GS_OK) return rc;
    if (group == GS_MASS) {
        k_get_grads<<<grid_for((size_t)m->E * m->N), 256, 0, st>>>(m->dev.gmass64, m->dev.perm_p, d_out, m->E, m->N);
    } else {
        const int t = group / 3, q = group % 3, c = m->counts[t];
        if (c == 0) return GS_OK;
        k_get_grads<<<grid_for((size_t)m->E * c), 256, 0, st>>>(m->dev.es[t].g64 + (size_t)q * m->E * c, m->dev.es[t].perm, d_out, m->E, c);
    }
    GS_LAUNCH_CHECK("k_get_grads");
    return GS_OK;
}
int launch_set_params(gs_model *m, int group, const float *d_values, cudaStream_t st) {
    if (group == GS_MASS) {
        k_set_params<<<grid_for((size_t)m->E * m->N), 256, 0, st>>>(m->d_inv_mass, m->dev.perm_p, d_values, m->E, m->N, 1);
    } else {
        const int t = group / 3, c = m->counts[t];
        if (c == 0) return GS_OK;
        k_set_params<<<grid_for((size_t)m->E * c), 256, 0, st>>>(m->d_param[group], m->dev.es[t].perm, d_values, m->E, c, 0);
    }
    GS_LAUNCH_CHECK("k_set_params");
    return GS_OK;
}

}  // namespace gs
