// gs_stream.cu -- the STREAMING plan: per substep one persistent element kernel and one particle kernel, forward
// and adjoint.
//
//   k_elements_fwd   persistent CTAs (SM count x co-resident CTAs) walk the Morton-ordered tiles of kTileElems
//                    elements: first their tets, then their triangles, then their hinges (all CTAs are in the same
//                    type's code at the same time, which keeps the instruction cache warm).  A tile's streams arrive
//                    through a double-buffered asynchronous pipeline: the tile's particle ids two tiles ahead and the
//                    gather list of its packed record one tile ahead by cp.async.bulk (TMA 1-D) signalling an
//                    mbarrier, issued by one thread; the particle states (x, v as float4) of the next tile by cp.async
//                    16 B per tile-particle from the ids already on chip; the thread-private record fields (16-bit
//                    staging indices, rest constants, material parameters) by a bulk L2 prefetch two tiles ahead and
//                    one coalesced register load per thread one tile ahead.  No thread waits on a dependent global
//                    load.  Tiles are dealt round-robin; the forward kernel claims its third and later tiles from a
//                    global queue.  One
//                    thread evaluates one element from shared memory, writes its per-vertex forces to conflict-free
//                    float4 slots; after one barrier every thread sums four consecutive entries of the tile's gather list
//                    (no shared-memory atomics: fp32 smem atomics are CAS loops on sm_100a) and issues ONE
//                    red.global.add.v4.f32 to the global force array.
//   k_particles_fwd  per particle: contact + friction from (x-, v-), semi-implicit Euler, writes the next tape
//                    slot, re-zeroes the force accumulator, flags non-finite states.
//   k_particles_adj  adjoint of integrate + contact; mass gradient; produces adj_f.
//   k_elements_adj   gather-form VJP of the element forces with the same tiles and pipeline (adj_f gathered too);
//                    parameter gradients leave as fire-and-forget red.global.add.f32.
//
// a1-a10 of SURVEY.md 8(a); citations of the formulas are in gs_elements.cuh.
#include <algorithm>
#include <climits>
#include <vector>

#include "gs_elements.cuh"
#include "gs_internal.h"

namespace gs {

#define GS_LAUNCH_CHECK(what)                                        \
    do {                                                             \
        cudaError_t e_ = cudaGetLastError();                         \
        if (e_ != cudaSuccess) return cuda_fail(e_, what);           \
        count_launch();                                              \
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
// the same, predicated: no branch, so the emit phase stays convergent
__device__ __forceinline__ void red_add_v4_if(unsigned pred, float4 *addr, float a, float b, float c) {
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %5, 0;\n\t@p red.global.add.v4.f32 [%0], {%1, %2, %3, %4};\n\t}" ::"l"(addr), "f"(a), "f"(b), "f"(c),
                 "f"(0.0f), "r"(pred)
                 : "memory");
}
// Segmented sum over a thread's 4 consecutive gather-list entries (sorted by tile-particle), branch-free.  Descriptor:
// bits 0-9 index of the first entry's particle in the tile's id list, bits 10-12 "entry k starts a new run" (k = 1..3),
// bits 13-15 number of valid entries.  Invalid entries point at slot 0 and are never flushed.
struct EmitPlan {
    unsigned s[4];       // slot of each entry
    unsigned fl;         // bit k: a run ends at entry k -> one reduction
    unsigned r[4];       // run number of entry k
    float keep[3];       // 0 if entry k+1 starts a new run, else 1
    const int *idp;
    __device__ __forceinline__ EmitPlan(uint2 sl, unsigned dsc, const int *ids) {
        const unsigned nv = dsc >> 13, bb = (dsc >> 10) & 7u;
        s[0] = sl.x & 0xFFFFu; s[1] = sl.x >> 16; s[2] = sl.y & 0xFFFFu; s[3] = sl.y >> 16;
        fl = bb | (1u << (nv - 1u));
        r[0] = 0u; r[1] = bb & 1u; r[2] = r[1] + ((bb >> 1) & 1u); r[3] = r[2] + (bb >> 2);
        keep[0] = (bb & 1u) ? 0.f : 1.f; keep[1] = (bb & 2u) ? 0.f : 1.f; keep[2] = (bb & 4u) ? 0.f : 1.f;
        idp = ids + (dsc & 1023u);
    }
    // checked build: every slot inside the output plane, every flushed run inside the tile's particle list with a valid id
    __device__ __forceinline__ bool in_range(int n_slots, int first, int pmax, int N) const {
        bool ok = (int)s[0] < n_slots && (int)s[1] < n_slots && (int)s[2] < n_slots && (int)s[3] < n_slots;
#pragma unroll
        for (int k = 0; k < 4; k++)
            if (fl & (1u << k)) ok = ok && first + (int)r[k] < pmax && idp[r[k]] >= 0 && idp[r[k]] < N;
        return ok;
    }
    // running sums a[k] of the runs; a[k] is final where bit k of fl is set
    __device__ __forceinline__ void sums(const float4 *src, float3 a[4]) const {
        const float4 c0 = src[s[0]], c1 = src[s[1]], c2 = src[s[2]], c3 = src[s[3]];
        a[0] = make_float3(c0.x, c0.y, c0.z);
        a[1] = make_float3(fmaf(a[0].x, keep[0], c1.x), fmaf(a[0].y, keep[0], c1.y), fmaf(a[0].z, keep[0], c1.z));
        a[2] = make_float3(fmaf(a[1].x, keep[1], c2.x), fmaf(a[1].y, keep[1], c2.y), fmaf(a[1].z, keep[1], c2.z));
        a[3] = make_float3(fmaf(a[2].x, keep[2], c3.x), fmaf(a[2].y, keep[2], c3.y), fmaf(a[2].z, keep[2], c3.z));
    }
    __device__ __forceinline__ void flush(float4 *dst, const float3 a[4]) const {
#pragma unroll
        for (int k = 0; k < 4; k++) red_add_v4_if(fl & (1u << k), dst + idp[r[k]], a[k].x, a[k].y, a[k].z);
    }
};
// Deterministic emit (gs_set_deterministic): as the plain emit, but a run of equal particles that crosses the 4-entry
// chunks of several threads is summed by the thread that owns its START, in entry order, and leaves as ONE reduction --
// the plain emit issues one per chunk, whose order at the L2 is not fixed.  A thread whose first run continues the previous
// thread's last run publishes that run's partial sum in `plane` (the output plane, free once every thread has read its
// entries: two extra CTA barriers); w = 1: the run ends inside the chunk, 2: the whole chunk belongs to the run.
// All threads of the CTA must call it.
__device__ __forceinline__ void emit_det(const uint16_t *slot_desc, const uint16_t *slots, const int *ids, float4 *plane, float4 *dst) {
    const int tid = threadIdx.x;
    const unsigned dsc = slot_desc[tid], nv = dsc >> 13;
    const bool has = nv > 0u;
    bool cont = false;
    if (has && tid > 0) {
        const unsigned dp = slot_desc[tid - 1];
        cont = (dp >> 13) > 0u && (dp & 1023u) + (unsigned)__popc((dp >> 10) & 7u) == (dsc & 1023u);
    }
    const EmitPlan ep(has ? reinterpret_cast<const uint2 *>(slots)[tid] : make_uint2(0u, 0u), has ? dsc : (1u << 13), ids);
    float3 a[4];
    ep.sums(plane, a);
    const int k0 = __ffs(ep.fl) - 1;  // entry at which my first run ends
    __syncthreads();
    plane[tid] = (has && cont) ? make_float4(a[k0].x, a[k0].y, a[k0].z, k0 == (int)nv - 1 ? 2.f : 1.f) : make_float4(0.f, 0.f, 0.f, 0.f);
    __syncthreads();
    if (!has) return;
#pragma unroll
    for (int k = 0; k < 4; k++) {
        if (!(ep.fl & (1u << k)) || (k == k0 && cont)) continue;
        float3 tot = a[k];
        if (k == (int)nv - 1)
            for (int u = tid + 1; u < kTileElems; u++) {
                const float4 c = plane[u];
                if (c.w == 0.f) break;
                tot.x += c.x; tot.y += c.y; tot.z += c.z;
                if (c.w != 2.f) break;
            }
        red_add_v4(dst + ep.idp[ep.r[k]], tot.x, tot.y, tot.z);
    }
}
__device__ __forceinline__ void red_add_f32(float *addr, float a) {
    asm volatile("red.global.add.f32 [%0], %1;" ::"l"(addr), "f"(a) : "memory");
}
__device__ __forceinline__ void red_add_f64(double *addr, double a) {
    asm volatile("red.global.add.f64 [%0], %1;" ::"l"(addr), "d"(a) : "memory");
}
// Programmatic dependent launch: the hot-path kernels are launched with programmatic stream serialization, so a kernel
// may start (and run its prologue: barrier init, bulk copies of STATIC tile data) while its predecessor drains.
// grid_dep_wait() blocks until the predecessor grid has completed and its writes are visible; nothing the predecessor
// produces may be touched before it.  Both are no-ops in a kernel launched without the attribute.
__device__ __forceinline__ void grid_dep_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void grid_dep_launch() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void cp_async16(void *smem_dst, const void *gmem_src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(smem_dst)), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }
// mbarrier + bulk async copy (TMA, 1-D): one thread arms the barrier with the byte count and issues the copy, the
// copy engine signals the barrier when the bytes have landed; every consumer thread waits on the phase parity
__device__ __forceinline__ void mbar_init(uint64_t *b, int count) { asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count) : "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t *b, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
// L2 policies: the static tile streams (records, parameters, particle lists: ~125 MB per pass on the 1M-tet scene, about
// the size of L2) are read once per launch -> evict_first, so that they do not push out the particle arrays (state, force
// and adjoint accumulators, ~8 MB each), which every tile re-reads and the next kernel needs -> evict_last.
__device__ __forceinline__ uint64_t l2_policy_evict_first() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ uint64_t l2_policy_evict_last() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ void bulk_g2s(void *smem_dst, const void *gmem_src, unsigned bytes, uint64_t *b, uint64_t policy) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(smem_u32(smem_dst)),
                 "l"(gmem_src), "r"(bytes), "r"(smem_u32(b)), "l"(policy)
                 : "memory");
}
__device__ __forceinline__ void bulk_prefetch_l2(const void *gmem_src, unsigned bytes, uint64_t policy) {
    asm volatile("cp.async.bulk.prefetch.L2.global.L2::cache_hint [%0], %1, %2;" ::"l"(gmem_src), "r"(bytes), "l"(policy) : "memory");
}
__device__ __forceinline__ void cp_async16_hint(void *smem_dst, const void *gmem_src, uint64_t policy) {
    asm volatile("cp.async.cg.shared.global.L2::cache_hint [%0], [%1], 16, %2;" ::"r"(smem_u32(smem_dst)), "l"(gmem_src), "l"(policy) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *b, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(b)),
        "r"(parity)
        : "memory");
}

// Checked build (python -m paper_2104_02646_b200.build --checked, -DGS_CHECKED): every index the tile pipeline takes from
// the packed tile data is range-checked before use; a violation raises the model's flag with a code >= kCheckBase (reported
// by gs_check_finite as "substep" kCheckBase + code) and the access is skipped.  compute-sanitizer is not available on this
// pool, so the GPU parity tests are run once against this build instead (profiles/r2_sanitizers.md).
constexpr int kCheckBase = 0x7e000000;
#ifdef GS_CHECKED
#define GS_CHECK_IDX(cond, code, md_bad) ((cond) ? true : (atomicMin((md_bad), kCheckBase + (code)), false))
#else
#define GS_CHECK_IDX(cond, code, md_bad) (true)
#endif

// ------------------------------------------------------------------------------------------ tile pipeline
// Shared memory of one CTA of a tile kernel (ADJ adds the gathered adj_f and a second output plane):
//   ids   int[3][pmax]                      particle ids of tiles i, i+1, i+2      (bulk copy, two tiles ahead)
//   loc   uint16[2][pmax]                   staging index of each list entry       (same bulk copy; dead after the gather)
//   buf   [2] { x, (v), (a) float4[lmax];   gathered particle states               (cp.async 16 B, one tile ahead)
//               slots uint16[4][128], slot_desc uint16[128] }   the record's gather list (bulk copy, one tile ahead)
//   out   float4[arity][128] (x2 for ADJ with velocities)   per element-vertex contributions
//   bars  uint64[5] per element type: full[2], idfull[3]; one int for the tile-queue hand-over
// The rest of the record (connectivity, rest constants) and the parameters never enter shared memory: ElemRegs.
template <int TYPE, bool ADJ>
struct TileSmem {
    using R = RecLayout<TYPE>;
    static constexpr bool kHasV = TYPE != T_HINGE;
    static constexpr int kGather = 1 + (kHasV ? 1 : 0) + (ADJ ? 1 : 0);
    static constexpr int kPar = TYPE != T_HINGE ? kParBytes : 0;
    static constexpr int kEmitBytes = R::kBytes - R::oSlots;  // gather-list slots + run descriptors: the only record fields other threads read
    __host__ __device__ static int buf_bytes(int lmax) { return lmax * 16 * kGather + kEmitBytes; }
    __host__ __device__ static int out_bytes() { return R::kArityT * kTileElems * 16 * ((ADJ && kHasV) ? 2 : 1); }
    __host__ __device__ static int total_bytes(int pmax, int lmax) { return 3 * pmax * 4 + 2 * pmax * 2 + 2 * buf_bytes(lmax) + out_bytes(); }
};

template <int TYPE, bool ADJ>
struct TileView {
    using R = RecLayout<TYPE>;
    using S = TileSmem<TYPE, ADJ>;
    float4 *x, *v, *a;
    char *emit;
    const uint16_t *slots, *slot_desc;
    __device__ __forceinline__ TileView(char *base, int lmax) {
        char *p = base;
        x = (float4 *)p; p += lmax * 16;
        v = (float4 *)p; if (S::kHasV) p += lmax * 16;
        a = (float4 *)p; if (ADJ) p += lmax * 16;
        emit = p;
        slots = (const uint16_t *)p;
        slot_desc = (const uint16_t *)(p + (R::oSlotDesc - R::oSlots));
    }
};

// The record fields only the owning thread reads (connectivity as staging indices, rest constants, material
// parameters) never pass through shared memory: each thread loads its own, coalesced, one tile ahead, into registers.
template <int TYPE>
struct ElemRegs {
    uint2 li;  // four 16-bit staging indices, unpacked only when the element is evaluated (keeps the load in flight)
    float4 c0, c1;
    float2 c2;
    float area, mu, lam, damp;
    float act;  // this substep's actuation of the element (0 = passive)
};

// The persistent tile loop shared by the forward and adjoint kernels.  `compute(tv, tile, env, e_local)` evaluates one
// element into the output slots; `emit(id, env, sums...)` is called once per tile-particle with its summed slots.
// ACT: the EXTENDED kernels: activation schedules and / or the lift / drag of the air on triangles
// (PAPER.md:586), each checked at run time inside; the plain kernels (ACT = false) carry neither.
// ME: the model has more than one environment (work item = tile x environment).  The single-environment kernels (the large
// meshes) carry none of the item -> (tile, env) divisions and environment offsets.
template <int TYPE, bool ADJ, bool ACT, bool ME>
struct TilePipe {
    using S = TileSmem<TYPE, ADJ>;
    const ElemDev &es;
    const int N, E, pmax, lmax, bb;
    int *idbuf;         // [3][pmax] particle ids of tiles i, i+1, i+2
    uint16_t *locbuf;   // [2][pmax] tile-local staging index of each list entry (only live between load and gather)
    char *bufs;
    float4 *out;
    uint64_t *bars;  // full[0..1], idfull[0..2]
    const float4 *x4, *v4, *a4;
    const float *act;  // [E][cpad] actuation of this substep for this element type, or null
    int *bad;          // the model's flag (checked build)
    uint64_t pol_stream, pol_keep;
    __device__ __forceinline__ TilePipe(const ModelDev &md, char *smem, uint64_t *bars_, const float4 *x4_, const float4 *v4_, const float4 *a4_, const float *act_)
        : es(md.es[TYPE]), N(md.N), E(md.E), pmax(md.es[TYPE].pmax), lmax(md.es[TYPE].lmax), bb(S::buf_bytes(md.es[TYPE].lmax)), bars(bars_), x4(x4_), v4(v4_), a4(a4_), act(act_), bad(md.bad) {
        idbuf = (int *)smem;
        locbuf = (uint16_t *)(smem + 3 * pmax * 4);
        bufs = smem + 3 * pmax * 4 + 2 * pmax * 2;
        out = (float4 *)(bufs + 2 * bb);
        pol_stream = l2_policy_evict_first();
        pol_keep = l2_policy_evict_last();
    }
    // work item -> (tile, env); single-environment models (the large meshes) skip the division
    // tiles this launch walks per environment: all of them, or (extended kernels, deterministic mode) one colour class
    __device__ __forceinline__ int n_walk() const { return (ACT && es.det_list) ? es.det_n : es.n_tiles; }
    __device__ __forceinline__ void split(int item, unsigned &tile, unsigned &env) const {
        if (!ME) { tile = (unsigned)item; env = 0u; }
        else { const unsigned nw = (unsigned)n_walk(); env = (unsigned)item / nw; tile = (unsigned)item - env * nw; }
        if (ACT && es.det_list) tile = (unsigned)es.det_list[tile];
    }
    // ids of the CTA's j-th item go to id buffer `slot` = j % 3, its staging indices to loc buffer `par` = j % 2
    __device__ __forceinline__ void load_ids(int item, int slot, int par) {  // one thread
        unsigned tile, env;
        split(item, tile, env);
        const char *blk = (const char *)es.tile_parts + (size_t)tile * pmax * 6;
        mbar_expect_tx(bars + 2 + slot, pmax * 6);
        bulk_g2s(idbuf + slot * pmax, blk, pmax * 4, bars + 2 + slot, pol_stream);
        bulk_g2s(locbuf + par * pmax, blk + pmax * 4, pmax * 2, bars + 2 + slot, pol_stream);
    }
    // The producer work of a tile is dealt to lane 0 of three different warps (load_ids: warp 0, the gather-list copy:
    // warp 1, the L2 prefetches: warp 2), so that no warp is a tile's worth of issue slots behind the others at the barrier.
    __device__ __forceinline__ void load_static(int item, int b) {  // one thread
        unsigned tile, env;
        split(item, tile, env);
        TileView<TYPE, ADJ> tv(bufs + b * bb, lmax);
        const char *rec = es.rec + (size_t)tile * es.rec_bytes;
        mbar_expect_tx(bars + b, S::kEmitBytes);
        bulk_g2s(tv.emit, rec + S::R::oSlots, S::kEmitBytes, bars + b, pol_stream);
    }
    __device__ __forceinline__ void prefetch_static(int item) {  // one thread
        unsigned tile, env;
        split(item, tile, env);
        const char *rec = es.rec + (size_t)tile * es.rec_bytes;
        // the thread-private part of the record goes to L2 now and to registers (load_regs) one tile later
        bulk_prefetch_l2(rec, S::R::oSlots, pol_stream);
        if (S::kPar) bulk_prefetch_l2(es.par + ((size_t)env * es.n_tiles + tile) * (3 * kTileElems), S::kPar, pol_stream);
    }
    __device__ __forceinline__ void load_regs(int item, ElemRegs<TYPE> &er) const {  // all threads
        unsigned tile, env;
        split(item, tile, env);
        const char *rec = es.rec + (size_t)tile * es.rec_bytes;
        const int tid = threadIdx.x;
        er.li = __ldcs((const uint2 *)(rec + S::R::oLidx) + tid);
        er.c0 = __ldcs((const float4 *)(rec + S::R::oC0) + tid);
        if (TYPE == T_TET) {
            er.c1 = __ldcs((const float4 *)(rec + S::R::oC1) + tid);
            er.c2 = __ldcs((const float2 *)(rec + S::R::oC2) + tid);
        }
        if (TYPE == T_TRI) er.area = __ldcs((const float *)(rec + S::R::oArea) + tid);
        if (S::kPar) {
            const float *q = es.par + ((size_t)env * es.n_tiles + tile) * (3 * kTileElems) + tid;
            er.mu = __ldcs(q); er.lam = __ldcs(q + kTileElems); er.damp = __ldcs(q + 2 * kTileElems);
        }
        er.act = (ACT && TYPE != T_TRI && act) ? __ldcs(act + ((size_t)env * es.n_tiles + tile) * kTileElems + tid) : 0.0f;
    }
    __device__ __forceinline__ void gather(int item, int slot, int b) {  // all threads
        unsigned tile, env;
        split(item, tile, env);
        TileView<TYPE, ADJ> tv(bufs + b * bb, lmax);
        const int *ids = idbuf + slot * pmax;
        const uint16_t *loc = locbuf + (b & 1) * pmax;  // the tile staged into buffer b is the CTA's item with parity b
        const size_t eoff = (size_t)env * N;
        for (int p = threadIdx.x; p < pmax; p += kTileElems) {
            const int id = ids[p];
            if (id >= 0) {
                const int l = loc[p];
                if (!GS_CHECK_IDX(id < N && l < lmax, 1, bad)) continue;
                cp_async16_hint(tv.x + l, x4 + eoff + id, pol_keep);
                if (S::kHasV) cp_async16_hint(tv.v + l, v4 + eoff + id, pol_keep);
                if (ADJ) cp_async16_hint(tv.a + l, a4 + eoff + id, pol_keep);
            }
        }
        cp_async_commit();
    }
    // `rot` = number of items of the types already walked: the round-robin deal of items to CTAs continues across the
    // types of one launch, so their remainders do not pile onto the same CTAs
    template <class Compute, class Emit>
    __device__ __forceinline__ void run_static(int rot, Compute compute, Emit emit) {
        const int n_items = n_walk() * E, G = gridDim.x, tid = threadIdx.x;
        const int first = (int)((blockIdx.x + (unsigned)G - (unsigned)rot % (unsigned)G) % (unsigned)G);  // item j of this type -> CTA (j + rot) mod G
        if (first >= n_items) return;
        const int cnt = (n_items - first + G - 1) / G;
        if (tid == 0) {
            load_ids(first, 0, 0);
            if (cnt > 1) load_ids(first + G, 1, 1);
        }
        if (tid == 32) load_static(first, 0);
        if (tid == 64) prefetch_static(first);
        ElemRegs<TYPE> er;
        load_regs(first, er);
        mbar_wait(bars + 2, 0);
        grid_dep_wait();  // the particle arrays gathered from here on are the predecessor kernel's output
        gather(first, 0, 0);
        int s3 = 0, q3 = 0;  // i % 3, i / 3: ids of the CTA's j-th item use id buffer j % 3 for the (j / 3)-th time
        for (int i = 0; i < cnt; i++) {
            const int item = first + i * G;
            const int s3n = s3 == 2 ? 0 : s3 + 1, s3nn = s3n == 2 ? 0 : s3n + 1;
            cp_async_wait_all();
            mbar_wait(bars + (i & 1), (i >> 1) & 1);
            if (i + 1 < cnt) mbar_wait(bars + 2 + s3n, (q3 + (s3n == 0 ? 1 : 0)) & 1);
            __syncthreads();
            if (tid == 0 && i + 2 < cnt) load_ids(item + 2 * G, s3nn, i & 1);
            if (tid == 32 && i + 1 < cnt) load_static(item + G, (i + 1) & 1);
            if (tid == 64 && i + 1 < cnt) prefetch_static(item + G);
            if (i + 1 < cnt) gather(item + G, s3n, (i + 1) & 1);
            unsigned tile, env;
            split(item, tile, env);
            const TileView<TYPE, ADJ> tv(bufs + (i & 1) * bb, lmax);
            if ((int)(tile * kTileElems + tid) < es.count) compute(tv, er, (int)tile, (int)env, out);
            if (i + 1 < cnt) load_regs(item + G, er);  // in flight across the barrier, the emit phase and the next waits
            __syncthreads();
            const int *ids = idbuf + s3 * pmax;
            emit(tv, ids, (int)env, out);
            if (s3n == 0) q3++;
            s3 = s3n;
        }
    }
    // Work distribution.  Forward kernel (kQueue): the CTA's first two items are static, (blockIdx + rot) mod G and that
    // + G (`rot` rotates the types of one launch against each other); every further item is claimed from the type's
    // global queue (`ctr`, zero at launch) by thread 0, one iteration before its particle ids are requested, i.e. three
    // tiles ahead of its evaluation, so the atomic's round trip is never waited on.  The queue evens out the tail of the
    // persistent grid (config 4 forward: -6 %).  Adjoint kernel: static stride G throughout -- with the queue the
    // compiler's register allocation tips from 80 to 96 registers (6 -> 5 CTAs per SM) and the kernel loses 5 %.
    static constexpr bool kQueue = !ADJ;
    template <class Compute, class Emit>
    __device__ __forceinline__ void run(int rot, int *ctr, int *next_slot, Compute compute, Emit emit) {
        if (!kQueue) { run_static(rot, compute, emit); return; }
        const int n_items = n_walk() * E, G = gridDim.x, tid = threadIdx.x;
        const int first = (int)((blockIdx.x + (unsigned)G - (unsigned)rot % (unsigned)G) % (unsigned)G);  // item j of this type -> CTA (j + rot) mod G
        if (first >= n_items) return;
        // otherwise the static items cover everything; the deterministic mode launches several times per substep between
        // two resets of the queue counters, so it deals statically
        const bool queue = kQueue && 2 * G < n_items && !(ACT && es.det_list);
        int item = first, item_n = first + G;  // items i, i+1 (all threads)
        int claimed = n_items;                 // kQueue: item i+2, thread 0 only until published through next_slot
        int ticket = -1;                       // raw result of the queue's atomicAdd for item i+3 (< 0: none): converted one
                                               // iteration later, so that the atomic's round trip is not waited on
        if (tid == 0) {
            load_ids(first, 0, 0);
            if (item_n < n_items) load_ids(item_n, 1, 1);
        }
        if (tid == 32) load_static(first, 0);
        if (tid == 64) prefetch_static(first);
        ElemRegs<TYPE> er;
        load_regs(first, er);
        mbar_wait(bars + 2, 0);
        grid_dep_wait();  // the particle arrays gathered from here on are the predecessor kernel's output
        if (kQueue && tid == 0 && queue) claimed = 2 * G + atomicAdd(ctr, 1);
        gather(first, 0, 0);
        int s3 = 0, q3 = 0;  // i % 3, i / 3: ids of the CTA's j-th item use id buffer j % 3 for the (j / 3)-th time
        for (int i = 0;; i++) {
            const int s3n = s3 == 2 ? 0 : s3 + 1, s3nn = s3n == 2 ? 0 : s3n + 1;
            const bool has_n = item_n < n_items;
            cp_async_wait_all();
            mbar_wait(bars + (i & 1), (i >> 1) & 1);
            if (has_n) mbar_wait(bars + 2 + s3n, (q3 + (s3n == 0 ? 1 : 0)) & 1);
            __syncthreads();
            if (tid == 0) {
                const int item_nn = kQueue ? claimed : item_n + G;  // item i+2
                if (kQueue) *next_slot = claimed;                   // read by everybody after the next barrier
                if (has_n && item_nn < n_items) load_ids(item_nn, s3nn, i & 1);
                if (kQueue) claimed = (queue && claimed < n_items) ? 2 * G + atomicAdd(ctr, 1) : n_items;  // item i+3
            }
            if (tid == 32 && has_n) load_static(item_n, (i + 1) & 1);
            if (tid == 64 && has_n) prefetch_static(item_n);
            if (has_n) gather(item_n, s3n, (i + 1) & 1);
            unsigned tile, env;
            split(item, tile, env);
            const TileView<TYPE, ADJ> tv(bufs + (i & 1) * bb, lmax);
            if ((int)(tile * kTileElems + tid) < es.count) compute(tv, er, (int)tile, (int)env, out);
            if (has_n) load_regs(item_n, er);  // in flight across the barrier, the emit phase and the next waits
            __syncthreads();
            const int *ids = idbuf + s3 * pmax;
            emit(tv, ids, (int)env, out);
            if (!has_n) break;
            item = item_n;
            item_n = kQueue ? *next_slot : item_n + G;
            if (s3n == 0) q3++;
            s3 = s3n;
        }
    }
};

template <bool ACT>
__device__ __forceinline__ int walked(const ElemDev &es) { return (ACT && es.det_list) ? es.det_n : es.n_tiles; }

// ------------------------------------------------------------------------------------------ forward elements
constexpr int kBarBytes = 128;  // 15 mbarriers at the start of shared memory (5 per element type) + the queue hand-over slot

__device__ __forceinline__ void init_barriers(uint64_t *bars) {
    if (threadIdx.x < 15) {  // one barrier per lane of the first warp: one instruction instead of 15 in a row
        mbar_init(bars + threadIdx.x, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
}

template <int TYPE, bool ACT, bool ME>
__device__ __forceinline__ void tiles_fwd(const ModelDev &md, const ActDev &ad, char *smem, uint64_t *bars, int *next_slot, int rot, const float4 *__restrict__ x4,
                                          const float4 *__restrict__ v4, float4 *__restrict__ f4) {
    const float *actp = TYPE == T_TET ? ad.tet : (TYPE == T_HINGE ? ad.hinge : nullptr);
    TilePipe<TYPE, false, ACT, ME> pipe(md, smem, bars, x4, v4, nullptr, actp);
    const int N = md.N;
    pipe.run(
        rot, md.tile_ctr + TYPE, next_slot,
        [&](const TileView<TYPE, false> &tv, const ElemRegs<TYPE> &er, int, int env, float4 *sf) {
            const int tid = threadIdx.x;
            const ushort4 li = make_ushort4((unsigned short)(er.li.x & 0xFFFFu), (unsigned short)(er.li.x >> 16), (unsigned short)(er.li.y & 0xFFFFu), (unsigned short)(er.li.y >> 16));
            if (!GS_CHECK_IDX(li.x < pipe.lmax && li.y < pipe.lmax && li.z < pipe.lmax && (TYPE == T_TRI || li.w < pipe.lmax), 2, md.bad)) return;
            if (TYPE == T_TET) {
                const float4 c0 = er.c0, c1 = er.c1;
                const float2 c2 = er.c2;
                const float b[9] = {c0.x, c0.y, c0.z, c0.w, c1.x, c1.y, c1.z, c1.w, c2.x};
                const vec3 x[4] = {vec3(tv.x[li.x]), vec3(tv.x[li.y]), vec3(tv.x[li.z]), vec3(tv.x[li.w])};
                const vec3 v[4] = {vec3(tv.v[li.x]), vec3(tv.v[li.y]), vec3(tv.v[li.z]), vec3(tv.v[li.w])};
                vec3 f[4];
                tet_force(x, v, b, c2.y, er.mu, er.lam, er.damp, er.act, f);
#pragma unroll
                for (int k = 0; k < 4; k++) sf[k * kTileElems + tid] = make_float4(f[k].x, f[k].y, f[k].z, 0.f);
            } else if (TYPE == T_TRI) {
                const float4 c0 = er.c0;
                const float b[4] = {c0.x, c0.y, c0.z, c0.w};
                const vec3 x[3] = {vec3(tv.x[li.x]), vec3(tv.x[li.y]), vec3(tv.x[li.z])};
                const vec3 v[3] = {vec3(tv.v[li.x]), vec3(tv.v[li.y]), vec3(tv.v[li.z])};
                vec3 f[3];
                tri_force(x, v, b, er.area, er.mu, er.lam, er.damp, f);
                if (ACT && md.aero) aero_force_add(x, v, vec3(md.wx, md.wy, md.wz), md.kdrag[env], md.klift[env], f);
#pragma unroll
                for (int k = 0; k < 3; k++) sf[k * kTileElems + tid] = make_float4(f[k].x, f[k].y, f[k].z, 0.f);
            } else {
                const float4 c0 = er.c0;
                const vec3 x[4] = {vec3(tv.x[li.x]), vec3(tv.x[li.y]), vec3(tv.x[li.z]), vec3(tv.x[li.w])};
                vec3 f[4];
                float sa = 0.0f, ca = 1.0f;
                if (ACT && actp) sincosf(er.act, &sa, &ca);
                hinge_force(x, c0.x, c0.y, c0.z, sa, ca, f);
#pragma unroll
                for (int k = 0; k < 4; k++) sf[k * kTileElems + tid] = make_float4(f[k].x, f[k].y, f[k].z, 0.f);
            }
        },
        [&](const TileView<TYPE, false> &tv, const int *ids, int env, const float4 *sf) {
            // thread t sums gather-list entries 4t .. 4t+3 (sorted by tile-particle) and issues one vector reduction per
            // run of equal particles: balanced over all lanes, no loop, no branch, no shared-memory atomics
            if (ACT && md.es[TYPE].det_list) { emit_det(tv.slot_desc, tv.slots, ids, const_cast<float4 *>(sf), f4 + (size_t)env * N); return; }
            const unsigned dsc = tv.slot_desc[threadIdx.x];
            if ((dsc >> 13) == 0u) return;
            const EmitPlan ep(reinterpret_cast<const uint2 *>(tv.slots)[threadIdx.x], dsc, ids);
            if (!GS_CHECK_IDX(ep.in_range(RecLayout<TYPE>::kArityT * kTileElems, (int)(dsc & 1023u), pipe.pmax, N), 3, md.bad)) return;
            float3 a[4];
            ep.sums(sf, a);
            ep.flush(f4 + (size_t)env * N, a);
        });
}

// all element types of one substep in ONE persistent launch: a CTA walks its tets, then its triangles, then its
// hinges (forces only meet in the global accumulator, so no grid-wide ordering is needed between the types)
template <bool ACT, bool ME>
__global__ void __launch_bounds__(kTileElems, 9) k_elements_fwd(const ModelDev md, const ActDev ad, const float4 *__restrict__ x4, const float4 *__restrict__ v4,
                                                             float4 *__restrict__ f4) {
    extern __shared__ __align__(16) char smem[];
    uint64_t *bars = (uint64_t *)smem;
    init_barriers(bars);
    int rot = 0;
    if (md.es[T_TET].count) { tiles_fwd<T_TET, ACT, ME>(md, ad, smem + kBarBytes, bars, (int *)(smem + 120), rot, x4, v4, f4); rot += walked<ACT>(md.es[T_TET]) * md.E; __syncthreads(); }
    if (md.es[T_TRI].count) { tiles_fwd<T_TRI, ACT, ME>(md, ad, smem + kBarBytes, bars + 5, (int *)(smem + 120), rot, x4, v4, f4); rot += walked<ACT>(md.es[T_TRI]) * md.E; __syncthreads(); }
    if (md.es[T_HINGE].count) tiles_fwd<T_HINGE, ACT, ME>(md, ad, smem + kBarBytes, bars + 10, (int *)(smem + 120), rot, x4, v4, f4);
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
    grid_dep_launch();
    grid_dep_wait();
    if (blockIdx.x == 0 && threadIdx.x < 3) md.tile_ctr[threadIdx.x] = 0;  // the forward element kernel's tile queues
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
// frame_off >= 0: the caller-order [E][N][3] cotangent dL/dx of the state AFTER this substep starts frame_off floats into
// the frame array whose base is in md.frame_base[0]; < 0: none.
__global__ void __launch_bounds__(256) k_particles_adj(const ModelDev md, const float4 *__restrict__ x4, const float4 *__restrict__ v4,
                                                       const float4 *__restrict__ v4n, long long frame_off,
                                                       float4 *__restrict__ adjx, float4 *__restrict__ adjv, float4 *__restrict__ adjf) {
    const size_t total = (size_t)md.E * md.N;
    grid_dep_launch();
    grid_dep_wait();
    if (blockIdx.x == 0 && threadIdx.x < 3) md.tile_ctr[3 + threadIdx.x] = 0;  // the adjoint element kernel's tile queues
    const int lane = threadIdx.x & 31;
    const float *frame_cot = frame_off >= 0 ? md.frame_base[0] + frame_off : nullptr;
    // block-uniform trip count: the contact-parameter gradients are reduced with full-warp shuffles
    for (size_t base = (size_t)blockIdx.x * blockDim.x; base < total; base += (size_t)gridDim.x * blockDim.x) {
        const size_t i = base + threadIdx.x;
        float gp[4] = {0.f, 0.f, 0.f, 0.f}, gg[3] = {0.f, 0.f, 0.f};
        int env = -1;
        if (i < total) {
            env = (int)(i / md.N);
            const int id = (int)(i - (size_t)env * md.N);
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
                gg[0] = dt * lv.x; gg[1] = dt * lv.y; gg[2] = dt * lv.z;  // v+ = v + (f w + g) dt  =>  dL/dg += dt lv
            }
            contact_adjoint(contact_params(md, env), x, v, af, ax, av, gp);
            adjx[i] = make_float4(ax.x, ax.y, ax.z, 0.f);
            adjv[i] = make_float4(av.x, av.y, av.z, 0.f);
            adjf[i] = make_float4(af.x, af.y, af.z, 0.f);
        }
        // per-environment totals (north_star (4): reduce with warp shuffles): dL/d(k_e, k_d, k_f, mu_c) from the warps that
        // have a particle in contact, and -- only when the model was asked for it (gs_request_grads: the extra reductions
        // cost 12 % of this kernel on the 476k-particle scene) -- dL/dg = dt sum_i [w_i > 0] lv_i from every warp.  Warp sums
        // in fp32 (32 terms), then one fp64 reduction per value and warp into one of kConSlots slots per environment.
        const bool mine = gp[0] != 0.f || gp[1] != 0.f || gp[2] != 0.f || gp[3] != 0.f;
        const unsigned act = __ballot_sync(0xffffffffu, mine);
        const unsigned live = md.want_gravity ? __ballot_sync(0xffffffffu, env >= 0) : act;
        if (live) {
            const int env0 = __shfl_sync(0xffffffffu, env, __ffs(live) - 1);
            const bool uni = __all_sync(0xffffffffu, env < 0 || env == env0);  // false: the warp straddles two environments
            const int sl = blockIdx.x & (kConSlots - 1);
            if (uni) {
                double *slot = md.gacc + ((size_t)env0 * kConSlots + sl) * kAccVals;
                if (act) {
#pragma unroll
                    for (int q = 0; q < 4; q++) {
                        float t = gp[q];
                        for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
                        if (lane == 0 && t != 0.f) red_add_f64(slot + q, (double)t);
                    }
                }
                if (md.want_gravity) {
#pragma unroll
                    for (int q = 0; q < 3; q++) {
                        float t = gg[q];
                        for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
                        if (lane == 0 && t != 0.f) red_add_f64(slot + 4 + q, (double)t);
                    }
                }
            } else if (env >= 0) {
                double *slot = md.gacc + ((size_t)env * kConSlots + sl) * kAccVals;
#pragma unroll
                for (int q = 0; q < 4; q++)
                    if (gp[q] != 0.f) red_add_f64(slot + q, (double)gp[q]);
                if (md.want_gravity) {
#pragma unroll
                    for (int q = 0; q < 3; q++)
                        if (gg[q] != 0.f) red_add_f64(slot + 4 + q, (double)gg[q]);
                }
            }
        }
    }
}

// ------------------------------------------------------------------------------------------ adjoint elements
template <int TYPE, bool ACT, bool ME>
__device__ __forceinline__ void tiles_adj(const ModelDev &md, const ActDev &ad, char *smem, uint64_t *bars, int *next_slot, int rot, const float4 *__restrict__ x4,
                                          const float4 *__restrict__ v4, const float4 *__restrict__ adjf, float4 *__restrict__ adjx,
                                          float4 *__restrict__ adjv) {
    const float *actp = TYPE == T_TET ? ad.tet : (TYPE == T_HINGE ? ad.hinge : nullptr);
    float *gactp = TYPE == T_TET ? ad.g_tet : (TYPE == T_HINGE ? ad.g_hinge : nullptr);
    TilePipe<TYPE, true, ACT, ME> pipe(md, smem, bars, x4, v4, adjf, actp);
    const int N = md.N;
    constexpr int PL = RecLayout<TYPE>::kArityT * kTileElems;  // second output plane: adj_v contributions
    const ElemDev &es = md.es[TYPE];
    const size_t gstride = (size_t)md.E * es.cpad;
    pipe.run(
        rot, md.tile_ctr + 3 + TYPE, next_slot,
        [&](const TileView<TYPE, true> &tv, const ElemRegs<TYPE> &er, int tile, int env, float4 *so) {
            const int tid = threadIdx.x;
            const ushort4 li = make_ushort4((unsigned short)(er.li.x & 0xFFFFu), (unsigned short)(er.li.x >> 16), (unsigned short)(er.li.y & 0xFFFFu), (unsigned short)(er.li.y >> 16));
            if (!GS_CHECK_IDX(li.x < pipe.lmax && li.y < pipe.lmax && li.z < pipe.lmax && (TYPE == T_TRI || li.w < pipe.lmax), 2, md.bad)) return;
            if (TYPE == T_TET) {
                const float4 c0 = er.c0, c1 = er.c1;
                const float2 c2 = er.c2;
                const float b[9] = {c0.x, c0.y, c0.z, c0.w, c1.x, c1.y, c1.z, c1.w, c2.x};
                const vec3 x[4] = {vec3(tv.x[li.x]), vec3(tv.x[li.y]), vec3(tv.x[li.z]), vec3(tv.x[li.w])};
                const vec3 v[4] = {vec3(tv.v[li.x]), vec3(tv.v[li.y]), vec3(tv.v[li.z]), vec3(tv.v[li.w])};
                const vec3 a[4] = {vec3(tv.a[li.x]), vec3(tv.a[li.y]), vec3(tv.a[li.z]), vec3(tv.a[li.w])};
                vec3 ax[4], av[4];
                float gmu, glam, gk, ga;
                tet_adjoint(x, v, a, b, c2.y, er.mu, er.lam, er.damp, er.act, ax, av, gmu, glam, gk, ga);
                float *g = es.g32 + (size_t)env * es.cpad + tile * kTileElems + tid;
                red_add_f32(g, gmu); red_add_f32(g + gstride, glam); red_add_f32(g + 2 * gstride, gk);
                if (ACT && gactp) red_add_f32(gactp + (size_t)env * es.cpad + tile * kTileElems + tid, ga);
#pragma unroll
                for (int k = 0; k < 4; k++) {
                    so[k * kTileElems + tid] = make_float4(ax[k].x, ax[k].y, ax[k].z, 0.f);
                    so[PL + k * kTileElems + tid] = make_float4(av[k].x, av[k].y, av[k].z, 0.f);
                }
            } else if (TYPE == T_TRI) {
                const float4 c0 = er.c0;
                const float b[4] = {c0.x, c0.y, c0.z, c0.w};
                const vec3 x[3] = {vec3(tv.x[li.x]), vec3(tv.x[li.y]), vec3(tv.x[li.z])};
                const vec3 v[3] = {vec3(tv.v[li.x]), vec3(tv.v[li.y]), vec3(tv.v[li.z])};
                const vec3 a[3] = {vec3(tv.a[li.x]), vec3(tv.a[li.y]), vec3(tv.a[li.z])};
                vec3 ax[3], av[3];
                float gmu, glam, gk;
                tri_adjoint(x, v, a, b, er.area, er.mu, er.lam, er.damp, ax, av, gmu, glam, gk);
                float *g = es.g32 + (size_t)env * es.cpad + tile * kTileElems + tid;
                red_add_f32(g, gmu); red_add_f32(g + gstride, glam); red_add_f32(g + 2 * gstride, gk);
                if (ACT && md.aero) {  // the triangle's terms of dL/dk_drag, dL/dk_lift go to rows 3, 4 of its gradient block
                    float gd, gl;
                    aero_adjoint_add(x, v, a, vec3(md.wx, md.wy, md.wz), md.kdrag[env], md.klift[env], ax, av, gd, gl);
                    red_add_f32(g + 3 * gstride, gd); red_add_f32(g + 4 * gstride, gl);
                }
#pragma unroll
                for (int k = 0; k < 3; k++) {
                    so[k * kTileElems + tid] = make_float4(ax[k].x, ax[k].y, ax[k].z, 0.f);
                    so[PL + k * kTileElems + tid] = make_float4(av[k].x, av[k].y, av[k].z, 0.f);
                }
            } else {
                const float4 c0 = er.c0;
                const vec3 x[4] = {vec3(tv.x[li.x]), vec3(tv.x[li.y]), vec3(tv.x[li.z]), vec3(tv.x[li.w])};
                const vec3 a[4] = {vec3(tv.a[li.x]), vec3(tv.a[li.y]), vec3(tv.a[li.z]), vec3(tv.a[li.w])};
                vec3 ax[4];
                float gkb, ga, sa = 0.0f, ca = 1.0f;
                if (ACT && actp) sincosf(er.act, &sa, &ca);
                hinge_adjoint(x, a, c0.x, c0.y, c0.z, c0.w, sa, ca, ax, gkb, ga);
                red_add_f32(es.g32 + (size_t)env * es.cpad + tile * kTileElems + tid, gkb);
                if (ACT && gactp) red_add_f32(gactp + (size_t)env * es.cpad + tile * kTileElems + tid, ga);
#pragma unroll
                for (int k = 0; k < 4; k++) so[k * kTileElems + tid] = make_float4(ax[k].x, ax[k].y, ax[k].z, 0.f);
            }
        },
        [&](const TileView<TYPE, true> &tv, const int *ids, int env, const float4 *so) {
            if (ACT && md.es[TYPE].det_list) {
                emit_det(tv.slot_desc, tv.slots, ids, const_cast<float4 *>(so), adjx + (size_t)env * N);
                if (TYPE != T_HINGE) emit_det(tv.slot_desc, tv.slots, ids, const_cast<float4 *>(so) + PL, adjv + (size_t)env * N);
                return;
            }
            const unsigned dsc = tv.slot_desc[threadIdx.x];
            if ((dsc >> 13) == 0u) return;
            const EmitPlan ep(reinterpret_cast<const uint2 *>(tv.slots)[threadIdx.x], dsc, ids);
            if (!GS_CHECK_IDX(ep.in_range(RecLayout<TYPE>::kArityT * kTileElems, (int)(dsc & 1023u), pipe.pmax, N), 3, md.bad)) return;
            float3 a[4];
            ep.sums(so, a);
            ep.flush(adjx + (size_t)env * N, a);
            if (TYPE != T_HINGE) {
                ep.sums(so + PL, a);
                ep.flush(adjv + (size_t)env * N, a);
            }
        });
}

template <bool ACT, bool ME>
__global__ void __launch_bounds__(kTileElems) k_elements_adj(const ModelDev md, const ActDev ad, const float4 *__restrict__ x4, const float4 *__restrict__ v4,
                                                             const float4 *__restrict__ adjf, float4 *__restrict__ adjx, float4 *__restrict__ adjv) {
    extern __shared__ __align__(16) char smem[];
    uint64_t *bars = (uint64_t *)smem;
    init_barriers(bars);
    int rot = 0;
    if (md.es[T_TET].count) { tiles_adj<T_TET, ACT, ME>(md, ad, smem + kBarBytes, bars, (int *)(smem + 120), rot, x4, v4, adjf, adjx, adjv); rot += walked<ACT>(md.es[T_TET]) * md.E; __syncthreads(); }
    if (md.es[T_TRI].count) { tiles_adj<T_TRI, ACT, ME>(md, ad, smem + kBarBytes, bars + 5, (int *)(smem + 120), rot, x4, v4, adjf, adjx, adjv); rot += walked<ACT>(md.es[T_TRI]) * md.E; __syncthreads(); }
    if (md.es[T_HINGE].count) tiles_adj<T_HINGE, ACT, ME>(md, ad, smem + kBarBytes, bars + 10, (int *)(smem + 120), rot, x4, v4, adjf, adjx, adjv);
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
// out[env][perm[e]] = g64[env][e]; internal arrays have row stride `stride` (>= count)
__global__ void k_get_grads(const double *__restrict__ g64, const int *__restrict__ perm, float *__restrict__ out, int E, int count, int stride) {
    const size_t total = (size_t)E * count;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        const int env = (int)(i / count), e = (int)(i - (size_t)env * count);
        out[(size_t)env * count + perm[e]] = (float)g64[(size_t)env * stride + e];
    }
}
// out[env] = sum over the elements of one row of a per-element gradient block (the air coefficients: one value per environment)
__global__ void k_sum_grad_row(const double *__restrict__ row, float *__restrict__ out, int count, int stride) {
    __shared__ double red[32];
    const int env = blockIdx.x;
    double s = 0.0;
    for (int e = threadIdx.x; e < count; e += blockDim.x) s += row[(size_t)env * stride + e];
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); w++) t += red[w];
        out[env] = (float)t;
    }
}
// q < 0: dst is the [E][count] inverse-mass array; else dst is ElemDev::par and q the parameter (0 mu, 1 lambda, 2 damp)
__global__ void k_set_params(float *__restrict__ dst, const int *__restrict__ perm, const float *__restrict__ src, int E, int count, int n_tiles, int q, int *__restrict__ bad) {
    const size_t total = (size_t)E * count;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        const int env = (int)(i / count), e = (int)(i - (size_t)env * count);
        const float val = src[(size_t)env * count + perm[e]];
        // same preconditions as gs_model_create: finite values, mass > 0, lambda > 0 (alpha = 1 + 3 mu / (4 lambda)); a
        // violation leaves the old value in place and raises the non-finite flag with substep index 0 (gs_check_finite)
        const bool ok = fabsf(val) <= 3.0e38f && ((q != -1 && q != 1) || val > 0.f);
        if (!ok) { atomicMin(bad, 0); continue; }
        if (q < 0) { if (dst[i] != 0.f) dst[i] = 1.0f / val; }  // pinned particles stay pinned
        else dst[par_index(n_tiles, env, e, q)] = val;
    }
}

// per-environment totals (contact parameters, gravity): fold the slots of (env, q) into the master and clear them
__global__ void k_flush_contact(double *__restrict__ gacc, double *__restrict__ g64, int n, int zero_master) {
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const int env = i / kAccVals, q = i % kAccVals;
        double s = 0.0;
        for (int k = 0; k < kConSlots; k++) {
            double *p = gacc + ((size_t)env * kConSlots + k) * kAccVals + q;
            s += *p;
            *p = 0.0;
        }
        g64[i] = zero_master ? 0.0 : g64[i] + s;
    }
}
// out[env][0 .. cnt) = master values q0 .. q0 + cnt of every environment
__global__ void k_get_contact(const double *__restrict__ g64, float *__restrict__ out, int E, int q0, int cnt) {
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < E * cnt; i += gridDim.x * blockDim.x) out[i] = (float)g64[(i / cnt) * kAccVals + q0 + i % cnt];
}
__global__ void k_set_scalar(float *__restrict__ dst, const float *__restrict__ src, int E) {
    for (int env = blockIdx.x * blockDim.x + threadIdx.x; env < E; env += gridDim.x * blockDim.x) dst[env] = src[env];
}

// k_b is shared by all environments and lives in the hinge records as kl = k_b * l0 (c0.z; l0 in c0.w): row 0 of src
__global__ void k_set_hinge_kb(char *__restrict__ rec, int rec_bytes, const int *__restrict__ perm, const float *__restrict__ src, int count) {
    for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < count; e += gridDim.x * blockDim.x) {
        float4 *c0 = reinterpret_cast<float4 *>(rec + (size_t)(e / kTileElems) * rec_bytes + RecLayout<T_HINGE>::oC0) + (e % kTileElems);
        c0->z = src[perm[e]] * c0->w;
    }
}

// ------------------------------------------------------------------------------------------ host launches
static inline int grid_for(size_t n, int block = 256) {
    size_t g = (n + block - 1) / block;
    const size_t cap = 148 * 16;  // grid-stride beyond this
    return (int)(g < 1 ? 1 : (g > cap ? cap : g));
}

// particle kernels: at most ONE resident wave (8 CTAs of 256 threads per SM), the rest by the grid-stride loop -- a partial
// second wave costs a whole wave's latency
static inline int grid_particles(size_t n) {
    size_t g = (n + 255) / 256;
    const size_t cap = 148 * 8;  // measured on config 4 (476 k particles): caps of 4, 6, 12, 16 per SM are 0.1-0.4 ms per step slower
    return (int)(g < 1 ? 1 : (g > cap ? cap : g));
}

// launch with programmatic stream serialization (see grid_dep_wait)
template <class... KArgs, class... Args>
static cudaError_t launch_pdl(bool pdl, void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}

template <class K>
static int tile_kernel_setup(K kern, int smem, int *ctas_per_sm) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(ctas_per_sm, kern, kTileElems, smem);
    if (e != cudaSuccess) return cuda_fail(e, "tile kernel setup");
    if (*ctas_per_sm < 1) { set_error("tile kernel does not fit an SM (%d bytes of shared memory)", smem); return GS_EINVAL; }
    return GS_OK;
}

int configure_stream_kernels(gs_model *m) {
    int dev = 0, sms = 148;
    if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    m->n_sms = sms;
    const ElemDev *es = m->dev.es;
    int fwd = 0, adj = 0;
    long long items = 0;
    for (int t = 0; t < N_TYPES; t++) {
        if (m->counts[t] == 0) continue;
        const int pm = es[t].pmax, lm = es[t].lmax;
        const int f = t == T_TET ? TileSmem<T_TET, false>::total_bytes(pm, lm) : t == T_TRI ? TileSmem<T_TRI, false>::total_bytes(pm, lm) : TileSmem<T_HINGE, false>::total_bytes(pm, lm);
        const int a = t == T_TET ? TileSmem<T_TET, true>::total_bytes(pm, lm) : t == T_TRI ? TileSmem<T_TRI, true>::total_bytes(pm, lm) : TileSmem<T_HINGE, true>::total_bytes(pm, lm);
        fwd = fwd > f ? fwd : f;
        adj = adj > a ? adj : a;
        items = std::max(items, (long long)es[t].n_tiles * m->E);
    }
    m->elem_items = items;
    if (items == 0) return GS_OK;
    m->smem_fwd = fwd + kBarBytes;
    m->smem_adj = adj + kBarBytes;
    // the actuated variants are set up first: the occupancy the launches use is that of the passive kernels, the actuated
    // ones must fit the same grid (they use a few registers more; a persistent grid that is not co-resident is still correct)
    int occ_a = 0;
    int rc = GS_OK;
    if (m->E > 1) {
        rc = tile_kernel_setup(k_elements_fwd<true, true>, m->smem_fwd, &occ_a);
        if (rc == GS_OK) rc = tile_kernel_setup(k_elements_adj<true, true>, m->smem_adj, &occ_a);
        if (rc == GS_OK) rc = tile_kernel_setup(k_elements_fwd<false, true>, m->smem_fwd, &m->occ_fwd);
        if (rc == GS_OK) rc = tile_kernel_setup(k_elements_adj<false, true>, m->smem_adj, &m->occ_adj);
    } else {
        rc = tile_kernel_setup(k_elements_fwd<true, false>, m->smem_fwd, &occ_a);
        if (rc == GS_OK) rc = tile_kernel_setup(k_elements_adj<true, false>, m->smem_adj, &occ_a);
        if (rc == GS_OK) rc = tile_kernel_setup(k_elements_fwd<false, false>, m->smem_fwd, &m->occ_fwd);
        if (rc == GS_OK) rc = tile_kernel_setup(k_elements_adj<false, false>, m->smem_adj, &m->occ_adj);
    }
    // Programmatic dependent launch pays where a kernel is a few microseconds long (20k tets, 157 tiles: -9 % per substep
    // pair): the next kernel's CTAs are resident and past their prologue when the predecessor drains.  It is neutral
    // from 350 to 650 tiles and costs beyond (250k tets +2.5 %, 490k tets +5 %): CTAs that launch into whatever slots
    // free up first are placed unevenly over the SMs.  The rule keeps the launch attribute while the largest type has
    // at most two tiles per SM.
    m->pdl = items <= 2LL * sms;
    return rc;
}

// persistent grid: every SM gets its full set of co-resident CTAs, never more CTAs than the largest type has work items
static inline int tile_grid(const gs_model *m, int occ) {
    const long long cap = (long long)m->n_sms * occ;
    return (int)(m->elem_items < cap ? m->elem_items : cap);
}

// deterministic mode: point the model description at colour class c; returns the largest item count of a type in it
static long long det_class(const gs_model *m, int c, ModelDev &md) {
    long long items = 0;
    for (int t = 0; t < N_TYPES; t++) {
        if (!m->counts[t]) continue;
        md.es[t].det_list = m->d_det[t] + m->det_off[t][c];
        md.es[t].det_n = m->det_off[t][c + 1] - m->det_off[t][c];
        items = std::max(items, (long long)md.es[t].det_n * m->E);
    }
    return items;
}

// substep < 0: a single-substep call (gs_step_forward / gs_step_backward): the activation frame is the model's current
// one (gs_set_actuation_frame) and a non-finite state is reported as substep 0
int stream_step_forward(gs_model *m, const float4 *x, const float4 *v, float4 *xo, float4 *vo, int substep, cudaStream_t st) {
    const ActDev ad = m->act_for(substep < 0 ? m->act_cur * m->act_stride : substep);
    const int bad_idx = substep < 0 ? 0 : substep;
    if (m->elem_items > 0 && m->det) {
        // deterministic mode: one launch of the extended kernel per colour class of tiles
        auto kern = m->E > 1 ? k_elements_fwd<true, true> : k_elements_fwd<true, false>;
        for (int c = 0; c < m->det_colours; c++) {
            ModelDev md = m->dev;
            long long items = det_class(m, c, md);
            if (items == 0) continue;
            const long long cap = (long long)m->n_sms * m->occ_fwd;
            GS_TIMED(m, GS_K_ELEMENTS_FWD, st, "k_elements_fwd", launch_pdl(false, kern, (int)std::min(items, cap), kTileElems, m->smem_fwd, st, md, ad, x, v, m->d_f));
        }
    } else if (m->elem_items > 0) {
        const bool act = m->act_frames > 0 || m->dev.aero, me = m->E > 1;
        auto kern = act ? (me ? k_elements_fwd<true, true> : k_elements_fwd<true, false>) : (me ? k_elements_fwd<false, true> : k_elements_fwd<false, false>);
        GS_TIMED(m, GS_K_ELEMENTS_FWD, st, "k_elements_fwd", launch_pdl(m->pdl, kern, tile_grid(m, m->occ_fwd), kTileElems, m->smem_fwd, st, m->dev, ad, x, v, m->d_f));
    }
    GS_TIMED(m, GS_K_PARTICLES_FWD, st, "k_particles_fwd", launch_pdl(m->pdl, k_particles_fwd, grid_particles((size_t)m->E * m->N), 256, 0, st, m->dev, x, v, m->d_f, xo, vo, bad_idx));
    return GS_OK;
}

// adjoint of the substep whose start state is (x, v) and whose end velocity is v_next; cotangents live in
// m->d_adjx / m->d_adjv (updated in place); the frame cotangent at frame_off (caller order, < 0: none) is added to adj_x first.
int stream_step_adjoint(gs_model *m, const float4 *x, const float4 *v, const float4 *v_next, long long frame_off, int substep, cudaStream_t st) {
    const ActDev ad = m->act_for(substep < 0 ? m->act_cur * m->act_stride : substep);
    GS_TIMED(m, GS_K_PARTICLES_ADJ, st, "k_particles_adj",
             launch_pdl(m->pdl, k_particles_adj, grid_particles((size_t)m->E * m->N), 256, 0, st, m->dev, x, v, v_next, frame_off, m->d_adjx, m->d_adjv, m->d_adjf));
    if (m->elem_items > 0 && m->det) {
        auto kern = m->E > 1 ? k_elements_adj<true, true> : k_elements_adj<true, false>;
        for (int c = 0; c < m->det_colours; c++) {
            ModelDev md = m->dev;
            long long items = det_class(m, c, md);
            if (items == 0) continue;
            const long long cap = (long long)m->n_sms * m->occ_adj;
            GS_TIMED(m, GS_K_ELEMENTS_ADJ, st, "k_elements_adj",
                     launch_pdl(false, kern, (int)std::min(items, cap), kTileElems, m->smem_adj, st, md, ad, x, v, m->d_adjf, m->d_adjx, m->d_adjv));
        }
    } else if (m->elem_items > 0) {
        const bool act = m->act_frames > 0 || m->dev.aero, me = m->E > 1;
        auto kern = act ? (me ? k_elements_adj<true, true> : k_elements_adj<true, false>) : (me ? k_elements_adj<false, true> : k_elements_adj<false, false>);
        GS_TIMED(m, GS_K_ELEMENTS_ADJ, st, "k_elements_adj",
                 launch_pdl(m->pdl, kern, tile_grid(m, m->occ_adj), kTileElems, m->smem_adj, st, m->dev, ad, x, v, m->d_adjf, m->d_adjx, m->d_adjv));
    }
    if (++m->steps_since_flush >= kFlushEvery) return launch_flush_grads(m, st);
    return GS_OK;
}

// activation schedules: caller order [F][E][count] <-> internal [F][E][cpad] (padding stays 0).  dir 0: ext -> internal
// values; dir 1: internal gradients -> ext
__global__ void k_actuation_io(float *__restrict__ internal, float *__restrict__ ext, const int *__restrict__ perm, int F, int E, int count, int cpad, int dir) {
    const size_t total = (size_t)F * E * count;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        const size_t fe = i / count;
        const int e = (int)(i - fe * count);
        if (dir == 0) internal[fe * cpad + e] = ext[fe * count + perm[e]];
        else ext[fe * count + perm[e]] = internal[fe * cpad + e];
    }
}
// dL/d(theta0) = -1/2 sum_f dL/d(alpha_f): the rest angle enters sin((theta - theta0)/2 + alpha) as -theta0/2
__global__ void k_theta0_grads(const float *__restrict__ gact, const int *__restrict__ perm, float *__restrict__ out, int F, int E, int count, int cpad) {
    const size_t total = (size_t)E * count;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        const int env = (int)(i / count), e = (int)(i - (size_t)env * count);
        double s = 0.0;
        for (int f = 0; f < F; f++) s += (double)gact[((size_t)f * E + env) * cpad + e];
        out[(size_t)env * count + perm[e]] = (float)(-0.5 * s);
    }
}
// rest angles live in the hinge records as (sin(theta0/2), cos(theta0/2)) in c0.x, c0.y: row 0 of src
__global__ void k_set_hinge_theta0(char *__restrict__ rec, int rec_bytes, const int *__restrict__ perm, const float *__restrict__ src, int count) {
    for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < count; e += gridDim.x * blockDim.x) {
        float4 *c0 = reinterpret_cast<float4 *>(rec + (size_t)(e / kTileElems) * rec_bytes + RecLayout<T_HINGE>::oC0) + (e % kTileElems);
        const double h = 0.5 * (double)src[perm[e]];
        c0->x = (float)sin(h); c0->y = (float)cos(h);
    }
}
int launch_actuation_io(gs_model *m, int kind, const float *d_in, float *d_out, cudaStream_t st) {
    const int t = kind == 0 ? T_TET : T_HINGE, c = m->counts[t];
    if (c == 0) return GS_OK;
    const size_t n = (size_t)m->act_frames * m->E * c;
    if (d_in) k_actuation_io<<<grid_for(n), 256, 0, st>>>(m->d_act[kind], const_cast<float *>(d_in), m->dev.es[t].perm, m->act_frames, m->E, c, m->hes[t].cpad, 0);
    else k_actuation_io<<<grid_for(n), 256, 0, st>>>(m->d_gact[kind], d_out, m->dev.es[t].perm, m->act_frames, m->E, c, m->hes[t].cpad, 1);
    GS_LAUNCH_CHECK("k_actuation_io");
    return GS_OK;
}

__global__ void k_set_ptr(const float **slot, const float *p) { *slot = p; }
int launch_set_frame_base(gs_model *m, const float *d_frames, cudaStream_t st) {
    k_set_ptr<<<1, 1, 0, st>>>(m->dev.frame_base, d_frames);
    GS_LAUNCH_CHECK("k_set_ptr");
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
    for (int t = 0; t < N_TYPES; t++) {
        const size_t n = m->counts[t] ? kNumGrads[t] * (size_t)m->E * m->hes[t].cpad : 0;
        if (!n) continue;
        GS_TIMED(m, GS_K_OTHER, st, "k_flush", k_flush<<<grid_for(n), 256, 0, st>>>(m->dev.es[t].g32, m->dev.es[t].g64, n));
    }
    GS_TIMED(m, GS_K_OTHER, st, "k_flush", k_flush<<<grid_for((size_t)m->E * m->N), 256, 0, st>>>(m->dev.gmass32, m->dev.gmass64, (size_t)m->E * m->N));
    GS_TIMED(m, GS_K_OTHER, st, "k_flush_contact", k_flush_contact<<<grid_for((size_t)m->E * kAccVals), 256, 0, st>>>(m->dev.gacc, m->dev.gcon64, m->E * kAccVals, 0));
    return GS_OK;
}
int launch_zero_grads(gs_model *m, cudaStream_t st) {
    m->steps_since_flush = 0;
    for (int k = 0; k < 2; k++) {  // dL/d(activation) of every frame
        const int t = k == 0 ? T_TET : T_HINGE;
        if (m->act_frames <= 0 || !m->counts[t]) continue;
        cudaError_t e = cudaMemsetAsync(m->d_gact[k], 0, sizeof(float) * (size_t)m->act_frames * m->E * m->hes[t].cpad, st);
        if (e != cudaSuccess) return cuda_fail(e, "zero actuation gradients");
    }
    for (int t = 0; t < N_TYPES; t++) {
        const size_t n = m->counts[t] ? kNumGrads[t] * (size_t)m->E * m->hes[t].cpad : 0;
        if (!n) continue;
        GS_TIMED(m, GS_K_OTHER, st, "k_zero", k_zero<<<grid_for(n), 256, 0, st>>>(m->dev.es[t].g32, m->dev.es[t].g64, n));
    }
    GS_TIMED(m, GS_K_OTHER, st, "k_zero", k_zero<<<grid_for((size_t)m->E * m->N), 256, 0, st>>>(m->dev.gmass32, m->dev.gmass64, (size_t)m->E * m->N));
    GS_TIMED(m, GS_K_OTHER, st, "k_flush_contact", k_flush_contact<<<grid_for((size_t)m->E * kAccVals), 256, 0, st>>>(m->dev.gacc, m->dev.gcon64, m->E * kAccVals, 1));
    return GS_OK;
}
int launch_get_grads(gs_model *m, int group, float *d_out, cudaStream_t st) {
    int rc = launch_flush_grads(m, st);
    if (rc != GS_OK) return rc;
    if (group == GS_MASS) {
        k_get_grads<<<grid_for((size_t)m->E * m->N), 256, 0, st>>>(m->dev.gmass64, m->dev.perm_p, d_out, m->E, m->N, m->N);
    } else if (group >= GS_CONTACT_KE && group <= GS_CONTACT_MUC) {
        k_get_contact<<<grid_for((size_t)m->E), 256, 0, st>>>(m->dev.gcon64, d_out, m->E, group - GS_CONTACT_KE, 1);
    } else if (group == GS_GRAVITY) {
        k_get_contact<<<grid_for((size_t)m->E * 3), 256, 0, st>>>(m->dev.gcon64, d_out, m->E, 4, 3);
    } else if (group == GS_AERO_DRAG || group == GS_AERO_LIFT) {
        const int c = m->counts[T_TRI], cp = m->hes[T_TRI].cpad;
        if (c == 0) { cudaMemsetAsync(d_out, 0, sizeof(float) * m->E, st); return GS_OK; }
        k_sum_grad_row<<<m->E, 256, 0, st>>>(m->dev.es[T_TRI].g64 + (size_t)(group == GS_AERO_DRAG ? 3 : 4) * m->E * cp, d_out, c, cp);
    } else if (group == GS_HINGE_THETA0) {
        const int c = m->counts[T_HINGE];
        if (c == 0) return GS_OK;
        if (m->act_frames <= 0) { set_error("dL/d(theta0) is read from the hinge actuation gradients: attach an activation schedule first (gs_actuation_create; one zero frame is enough)"); return GS_ESTATE; }
        k_theta0_grads<<<grid_for((size_t)m->E * c), 256, 0, st>>>(m->d_gact[1], m->dev.es[T_HINGE].perm, d_out, m->act_frames, m->E, c, m->hes[T_HINGE].cpad);
    } else {
        const int t = group == GS_HINGE_KB ? T_HINGE : group / 3, q = group == GS_HINGE_KB ? 0 : group % 3, c = m->counts[t];
        if (c == 0) return GS_OK;
        k_get_grads<<<grid_for((size_t)m->E * c), 256, 0, st>>>(m->dev.es[t].g64 + (size_t)q * m->E * m->hes[t].cpad, m->dev.es[t].perm, d_out, m->E, c, m->hes[t].cpad);
    }
    GS_LAUNCH_CHECK("k_get_grads");
    return GS_OK;
}
int launch_set_params(gs_model *m, int group, const float *d_values, cudaStream_t st) {
    if (group == GS_AERO_DRAG || group == GS_AERO_LIFT) {
        // the extended kernels run iff some coefficient is non-zero: read the values back (synchronises the stream)
        std::vector<float> h(m->E);
        float *dst = const_cast<float *>(group == GS_AERO_DRAG ? m->dev.kdrag : m->dev.klift);
        const float *other = group == GS_AERO_DRAG ? m->dev.klift : m->dev.kdrag;
        cudaError_t e = cudaMemcpyAsync(h.data(), d_values, sizeof(float) * m->E, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) return cuda_fail(e, "read air coefficients");
        bool any = false;
        for (float q : h) {
            if (!(q >= 0.0f) || !(q <= 3.0e38f)) { set_error("k_drag / k_lift must be finite and >= 0"); return GS_EINVAL; }
            any = any || q != 0.0f;
        }
        std::vector<float> o(m->E);
        e = cudaMemcpyAsync(o.data(), other, sizeof(float) * m->E, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaMemcpyAsync(dst, d_values, sizeof(float) * m->E, cudaMemcpyDeviceToDevice, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) return cuda_fail(e, "set air coefficients");
        for (float q : o) any = any || q != 0.0f;
        const int aero = (any && m->counts[T_TRI] > 0) ? 1 : 0;
        if (aero != m->dev.aero) { m->dev.aero = aero; m->epoch++; }
        return GS_OK;
    }
    if (group == GS_GRAVITY || group == GS_WIND) {
        // gravity / wind are by-value kernel arguments (ModelDev): read the three floats back (synchronises the stream) and
        // bump the epoch so that tapes re-capture their graphs
        float g[3];
        cudaError_t e = cudaMemcpyAsync(g, d_values, sizeof g, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) return cuda_fail(e, "read gravity");
        if (!(fabsf(g[0]) <= 3.0e38f) || !(fabsf(g[1]) <= 3.0e38f) || !(fabsf(g[2]) <= 3.0e38f)) { set_error("gravity / wind must be finite"); return GS_EINVAL; }
        if (group == GS_GRAVITY) { m->dev.gx = g[0]; m->dev.gy = g[1]; m->dev.gz = g[2]; }
        else { m->dev.wx = g[0]; m->dev.wy = g[1]; m->dev.wz = g[2]; }
        m->epoch++;
        return GS_OK;
    }
    if (group == GS_MASS) {
        k_set_params<<<grid_for((size_t)m->E * m->N), 256, 0, st>>>(m->d_inv_mass, m->dev.perm_p, d_values, m->E, m->N, 0, -1, m->dev.bad);
    } else if (group >= GS_CONTACT_KE && group <= GS_CONTACT_MUC) {
        const float *dst[4] = {m->dev.ke, m->dev.kd, m->dev.kf, m->dev.muc};
        k_set_scalar<<<grid_for((size_t)m->E), 256, 0, st>>>(const_cast<float *>(dst[group - GS_CONTACT_KE]), d_values, m->E);
    } else if (group == GS_HINGE_THETA0) {
        const int c = m->counts[T_HINGE];
        if (c == 0) return GS_OK;
        k_set_hinge_theta0<<<grid_for((size_t)c), 256, 0, st>>>(const_cast<char *>(m->dev.es[T_HINGE].rec), m->dev.es[T_HINGE].rec_bytes, m->dev.es[T_HINGE].perm, d_values, c);
    } else if (group == GS_HINGE_KB) {
        const int c = m->counts[T_HINGE];
        if (c == 0) return GS_OK;
        k_set_hinge_kb<<<grid_for((size_t)c), 256, 0, st>>>(const_cast<char *>(m->dev.es[T_HINGE].rec), m->dev.es[T_HINGE].rec_bytes, m->dev.es[T_HINGE].perm, d_values, c);
    } else {
        const int t = group / 3, c = m->counts[t];
        if (c == 0) return GS_OK;
        k_set_params<<<grid_for((size_t)m->E * c), 256, 0, st>>>(m->dev.es[t].par, m->dev.es[t].perm, d_values, m->E, c, m->dev.es[t].n_tiles, group % 3, m->dev.bad);
    }
    GS_LAUNCH_CHECK("k_set_params");
    return GS_OK;
}

}  // namespace gs
