// Shared device helpers for the sm_100a kernels: PTX wrappers (mbarrier, TMA, tcgen05/TMEM),
// E4M3 conversion, rounding-controlled fp32 arithmetic.  No CUTLASS; plain inline PTX.
#pragma once
#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <cuda_fp8.h>
#include <cuda.h>
#include <stdint.h>

namespace ev {

// ---- fp32 arithmetic that the compiler may not contract into FMA (DESIGN.md "rounding points":
// element-wise ops are single IEEE fp32 operations in the order the method states) -------------
__device__ __forceinline__ float mul_rn(float a, float b) { return __fmul_rn(a, b); }
__device__ __forceinline__ float add_rn(float a, float b) { return __fadd_rn(a, b); }
__device__ __forceinline__ float sub_rn(float a, float b) { return __fsub_rn(a, b); }
__device__ __forceinline__ float div_rn(float a, float b) { return __fdiv_rn(a, b); }

// ---- E4M3: hardware round-to-nearest-even, saturate-to-finite (cvt.rn.satfinite.e4m3x2.f32) ----
__device__ __forceinline__ uint16_t e4m3x2(float lo, float hi) {
    return (uint16_t)__nv_cvt_float2_to_fp8x2(make_float2(lo, hi), __NV_SATFINITE, __NV_E4M3);
}
__device__ __forceinline__ uint32_t e4m3x4(float a, float b, float c, float d) {
    return (uint32_t)e4m3x2(a, b) | ((uint32_t)e4m3x2(c, d) << 16);
}

__device__ __forceinline__ float bf16_bits_to_float(uint16_t b) { return __uint_as_float(((uint32_t)b) << 16); }

// e^x for the softmax weights of the attention merge: one FMUL + one MUFU.EX2 (2 ulp), the approximation the tensor-core
// attention kernel uses for its own probabilities; deterministic (the same bits for the same input on every launch)
__device__ __forceinline__ float exp_fast(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x * 1.4426950408889634f));
    return y;
}

// ---- warp / block reductions ------------------------------------------------------------------
__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// ---- shared-memory address / mbarrier ---------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void fence_barrier_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}" ::"r"(smem_u32(bar)), "r"(parity)
        : "memory");
}

// ---- TMA (cp.async.bulk.tensor) ---------------------------------------------------------------
__device__ __forceinline__ void tma_prefetch_desc(const CUtensorMap* m) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(m) : "memory");
}
// 2-D tile load: c0 = innermost (contiguous) coordinate, c1 = row coordinate
__device__ __forceinline__ void tma_load_2d(void* smem_dst, const CUtensorMap* m, uint64_t* bar, int c0, int c1) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];" ::"r"(
            smem_u32(smem_dst)),
        "l"(m), "r"(smem_u32(bar)), "r"(c0), "r"(c1)
        : "memory");
}
__device__ __forceinline__ void tma_load_4d(void* smem_dst, const CUtensorMap* m, uint64_t* bar, int c0, int c1, int c2, int c3) {
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];" ::"r"(
            smem_u32(smem_dst)),
        "l"(m), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
        : "memory");
}
__device__ __forceinline__ void tma_load_2d_hint(void* smem_dst, const CUtensorMap* m, uint64_t* bar, int c0, int c1,
                                                 uint64_t policy) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%3, %4}], [%2], %5;" ::"r"(
            smem_u32(smem_dst)),
        "l"(m), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "l"(policy)
        : "memory");
}
__device__ __forceinline__ uint64_t policy_evict_first() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ uint64_t policy_evict_last() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    return p;
}

// ---- tcgen05 / TMEM ---------------------------------------------------------------------------
template <int NCOLS>
__device__ __forceinline__ void tmem_alloc(uint32_t* smem_result) {  // one full warp
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(smem_result)), "n"(NCOLS)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
template <int NCOLS>
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr) {  // same warp that allocated
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "n"(NCOLS) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

// D[tmem] (+)= A[smem] * B[smem]^T, E4M3 x E4M3 -> fp32; issued by ONE thread
__device__ __forceinline__ void umma_f8(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f8f6f4 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem),
        "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate)
        : "memory");
}
// all previously issued tcgen05.mma of this thread arrive on the mbarrier when complete
// KV pool containers.  K and V are ROUNDED to bf16 (the method's rounding point, DESIGN.md R-round).  A cache read by
// the tcgen05 attention kernel keeps those bf16 values in binary16 containers (same 2 bytes per element): kind::f16
// wants both MMA operands in one format and Q / P are split into fp16 parts.  bf16 -> fp16 is exact for
// 2^-17 <= |x| <= 65504, keeps 2^-25 absolute below, and saturates above (no inf can enter the pool).
__device__ __forceinline__ uint32_t bf16x2_to_f16x2(uint32_t w) {
    uint32_t r;
    asm("cvt.rn.satfinite.f16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(__uint_as_float(w & 0xFFFF0000u)), "f"(__uint_as_float(w << 16)));
    return r;
}
__device__ __forceinline__ uint32_t f16x2_to_bf16x2(uint32_t w) {   // exact for values that came from bf16
    float lo, hi;
    asm("{\n\t.reg .b16 l, h;\n\tmov.b32 {l, h}, %2;\n\tcvt.f32.f16 %0, l;\n\tcvt.f32.f16 %1, h;\n\t}" : "=f"(lo), "=f"(hi) : "r"(w));
    uint32_t r;
    asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
    return r;
}
__device__ __forceinline__ bool elect_one() {  // one lane of a converged warp
    uint32_t pred;
    asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(pred));
    return pred != 0;
}
__device__ __forceinline__ void umma_commit(uint64_t* bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// 32 lanes x 16 consecutive fp32 columns: thread t of the warp gets lane (base_lane + t)
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t* v) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
          "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
        : "r"(taddr)
        : "memory");
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// K-major operand tile in shared memory, 128-byte rows, SWIZZLE_128B (the layout TMA writes with
// CU_TENSOR_MAP_SWIZZLE_128B): 8-row groups are 1024 B apart (SBO), version 1, layout type 2.
__device__ __forceinline__ uint64_t umma_desc_k128(uint32_t smem_addr, uint32_t sbo = 1024) {
    uint64_t d = 0;
    d |= (uint64_t)((smem_addr & 0x3FFFFu) >> 4);  // start address, 16-B units
    d |= (uint64_t)1 << 16;                        // leading byte offset (unused for swizzled K-major)
    d |= (uint64_t)(sbo >> 4) << 32;               // stride byte offset
    d |= (uint64_t)1 << 46;                        // descriptor version (Blackwell)
    d |= (uint64_t)2 << 61;                        // SWIZZLE_128B
    return d;
}
// instruction descriptor, kind::f8f6f4: D fp32, A = B = E4M3, both K-major, M x N
__host__ __device__ constexpr uint32_t umma_idesc_e4m3(int M, int N) {
    return (1u << 4) | (0u << 7) | (0u << 10) | (0u << 15) | (0u << 16) | ((uint32_t)(N >> 3) << 17) |
           ((uint32_t)(M >> 4) << 24);
}

// ---- output of a W8A8 linear as its consumer sees it ------------------------------------------------
// The layer GEMMs write raw fp32 accumulators, one [M][ld] slab per K-split; the consumer forms
//   y[m][n] = (((p_0 + p_1) + ...) + p_{S-1}) * s_x[m] * s_w[n]        (fixed order: deterministic)
// with single rounded fp32 operations, exactly the epilogue the method defines (DESIGN.md R-accum).
struct LinOut {
    const float* p;      // [slabs][M][ld]
    int splits, ld;      // splits: uniform slab count (classic split-K), or the maximum (stream-K)
    long split_stride;   // M * ld
    const float* sx;     // [M]
    const float* sw;     // [N]
    int sk_G, sk_U, sk_kb;  // canonical K cuts (ev_gemm.cuh): CTA pairs, K-block units, K-blocks per tile; sk_U == 0 = no cuts
};
// number of slabs that hold a piece of output channel n (all channels of a PAIR of 128-row weight tiles share it)
__device__ __forceinline__ int lin_slabs(const LinOut& o, int n) {
    if (o.sk_U == 0) return o.splits;
    const unsigned t = (unsigned)n >> 8, G = (unsigned)o.sk_G, U = (unsigned)o.sk_U, kb = (unsigned)o.sk_kb;
    const unsigned c_first = ((t * kb + 1u) * G + U - 1u) / U;   // first CTA touching the tile, + 1
    const unsigned c_last = ((t + 1u) * kb * G + U - 1u) / U;    // last CTA touching it, + 1
    return (int)(c_last - c_first) + 1;
}
__device__ __forceinline__ float lin_acc(const LinOut& o, size_t idx, int n) {
    const int cnt = lin_slabs(o, n);
    float acc = __ldcg(o.p + idx);
    for (int s = 1; s < cnt; ++s) acc = __fadd_rn(acc, __ldcg(o.p + (size_t)s * o.split_stride + idx));
    return acc;
}
__device__ __forceinline__ float lin_value(const LinOut& o, int m, int n, float sxm) {
    return __fmul_rn(__fmul_rn(lin_acc(o, (size_t)m * o.ld + n, n), sxm), __ldg(o.sw + n));
}

// four consecutive channels n..n+3 (n % 4 == 0, ld % 4 == 0): 16-byte loads, all slabs in flight together.
// MAXS = compile-time bound of the slab count (o.splits <= MAXS): bounds the registers held for loads in flight.
template <int MAXS = 8>
__device__ __forceinline__ float4 lin_value4(const LinOut& o, int m, int n, float sxm) {
    const size_t idx = (size_t)m * o.ld + n;
    const int cnt = MAXS == 1 ? 1 : lin_slabs(o, n);
    float4 acc = __ldcg(reinterpret_cast<const float4*>(o.p + idx));
    float4 t[MAXS > 1 ? MAXS - 1 : 1];
#pragma unroll
    for (int s = 1; s < MAXS; ++s)
        if (s < cnt) t[s - 1] = __ldcg(reinterpret_cast<const float4*>(o.p + (size_t)s * o.split_stride + idx));
#pragma unroll
    for (int s = 1; s < MAXS; ++s)
        if (s < cnt) {
            acc.x = __fadd_rn(acc.x, t[s - 1].x); acc.y = __fadd_rn(acc.y, t[s - 1].y);
            acc.z = __fadd_rn(acc.z, t[s - 1].z); acc.w = __fadd_rn(acc.w, t[s - 1].w);
        }
    const float4 w = __ldg(reinterpret_cast<const float4*>(o.sw + n));
    return make_float4(__fmul_rn(__fmul_rn(acc.x, sxm), w.x), __fmul_rn(__fmul_rn(acc.y, sxm), w.y),
                       __fmul_rn(__fmul_rn(acc.z, sxm), w.z), __fmul_rn(__fmul_rn(acc.w, sxm), w.w));
}

// ---- programmatic dependent launch -----------------------------------------------------------------
// A kernel launched with the programmatic-serialization attribute may begin while its predecessor
// runs; it must execute pdl_wait() before touching anything the predecessor wrote.  A predecessor
// calls pdl_launch_dependents() as early as possible so the dependent's prologue overlaps it.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// ---- weight stream -> L2 ahead of use ---------------------------------------------------------------
// At small M the step is bound by streaming 7.5 GB of weights, but the chain of short dependent kernels
// between the GEMMs (norm, RoPE, attention, merge, SwiGLU) leaves HBM idle most of the time.  Every kernel
// of the step therefore carries one slice of the upcoming GEMMs' weights and, before griddepcontrol.wait,
// asks the L2 to fetch it (cp.async.bulk.prefetch.L2: fire and forget, no registers, no shared memory).
// The 126 MB L2 becomes the staging buffer of a continuous weight stream; the host (PfPlanner, ev_api.cu)
// bounds how far the stream may run ahead of the GEMM that is consuming it.
struct L2Prefetch {
    const uint8_t* p[2];   // up to two pieces (a slice may straddle two matrices); 16-byte aligned
    unsigned n[2];         // bytes, multiples of L2PF_CHUNK
    unsigned long long* trace;  // null, or this launch's TRACE_SLOTS step-trace slots (ev_profile_trace): min over CTAs of
                                // t_enter, t_past_wait, ~t_exit, ~t_past_wait (globaltimer ns; memset 0xFF = empty)
};
__device__ __forceinline__ void trace_mark(const L2Prefetch& pf, int slot, bool complement, unsigned tid = 0) {
    if (pf.trace && threadIdx.x == tid) {
        unsigned long long t;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
        atomicMin(pf.trace + slot, complement ? ~t : t);
    }
}
__device__ __forceinline__ void trace_past_wait(const L2Prefetch& pf, unsigned tid = 0) { trace_mark(pf, 1, false, tid); trace_mark(pf, 3, true, tid); }
__device__ __forceinline__ void trace_exit(const L2Prefetch& pf) { trace_mark(pf, 2, true); }
// bring-up: phase k (0..3) reached by the LAST CTA (slots 4..7 hold ~t)
__device__ __forceinline__ void trace_phase(const L2Prefetch& pf, int k) { trace_mark(pf, 4 + k, true); }
constexpr int TRACE_SLOTS = 8;
// same, from whichever thread calls (the caller selects one thread)
__device__ __forceinline__ void trace_phase_any(const L2Prefetch& pf, int k) {
    if (pf.trace) {
        unsigned long long t;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
        atomicMin(pf.trace + 4 + k, ~t);
    }
}
// same, but ordered after the instruction that produced `dep` (e.g. a load)
__device__ __forceinline__ void trace_phase_dep(const L2Prefetch& pf, int k, float dep) {
    if (pf.trace && threadIdx.x == 0) {
        unsigned long long t;
        asm volatile("{\n\t.reg .f32 d;\n\tmov.f32 d, %1;\n\tmov.u64 %0, %%globaltimer;\n\t}" : "=l"(t) : "f"(dep));
        atomicMin(pf.trace + 4 + k, ~t);
    }
}
constexpr unsigned L2PF_CHUNK = 8192;
__device__ __forceinline__ void l2_prefetch_issue(const L2Prefetch& pf, unsigned first_thread = 0) {
    trace_mark(pf, 0, false);
    const unsigned lane = threadIdx.x - first_thread;   // the 32 threads [first_thread, +32) issue
    if (lane >= 32u || (pf.n[0] | pf.n[1]) == 0) return;
    const unsigned cta = blockIdx.x + gridDim.x * (blockIdx.y + gridDim.y * blockIdx.z);
    const unsigned ncta = gridDim.x * gridDim.y * gridDim.z;
#pragma unroll
    for (int s = 0; s < 2; ++s) {
        const unsigned chunks = pf.n[s] / L2PF_CHUNK;
        for (unsigned i = cta * 32u + lane; i < chunks; i += ncta * 32u)
            asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(pf.p[s] + (size_t)i * L2PF_CHUNK), "r"(L2PF_CHUNK) : "memory");
    }
}

// ---- thread-block clusters: a token row of the element-wise kernels is spread over the CTAs of one cluster
// (so that M = 60 rows still occupy all SMs); row statistics meet through distributed shared memory.
// Push model: every CTA stores its value into slot [own rank] of every peer, one cluster barrier, then each CTA
// reads its own shared memory in rank order (deterministic).  A launch without the cluster attribute is a
// cluster of one CTA: the same code runs.
__device__ __forceinline__ uint32_t cluster_ctarank() { uint32_t r; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ uint32_t cluster_nctarank() { uint32_t r; asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ void cluster_barrier() {
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ uint32_t cluster_map(const void* local_smem, uint32_t rank) {
    uint32_t ra;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(ra) : "r"(smem_u32(local_smem)), "r"(rank));
    return ra;
}
constexpr int CLUSTER_MAX = 8;
// v: a value every thread of the CTA already holds (block-reduced); xch: CLUSTER_MAX slots of shared memory,
// used once per kernel.  All threads of all CTAs of the cluster must call.
__device__ __forceinline__ float cluster_max(float v, float* xch) {
    const uint32_t nct = cluster_nctarank();
    if (nct == 1) return v;
    if (threadIdx.x < nct) asm volatile("st.shared::cluster.f32 [%0], %1;" ::"r"(cluster_map(xch + cluster_ctarank(), threadIdx.x)), "f"(v) : "memory");
    cluster_barrier();
    float r = xch[0];
    for (uint32_t i = 1; i < nct; ++i) r = fmaxf(r, xch[i]);
    return r;
}
__device__ __forceinline__ double cluster_sum(double v, double* xch) {
    const uint32_t nct = cluster_nctarank();
    if (nct == 1) return v;
    if (threadIdx.x < nct) asm volatile("st.shared::cluster.f64 [%0], %1;" ::"r"(cluster_map(xch + cluster_ctarank(), threadIdx.x)), "d"(v) : "memory");
    cluster_barrier();
    double r = xch[0];
    for (uint32_t i = 1; i < nct; ++i) r += xch[i];
    return r;
}

// ---- cp.async (Ampere-style, for the paged KV gathers) ------------------------------------------
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(smem_dst)), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

}  // namespace ev
