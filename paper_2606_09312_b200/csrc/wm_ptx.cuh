// PTX wrappers shared by the tcgen05 kernels (wm_tc.cu: one CTA per tile; wm_tc2.cu: CTA pair per tile).
// mbarrier / bulk-copy / tcgen05 (alloc, mma, commit, ld, st) / descriptors.  sm_100a only.
#pragma once

#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <stdint.h>

#include <cstdio>

#include "wm_internal.h"

namespace wm {

// host: fp32 (a bf16 value) -> fp16 bits, round to nearest even; false when the value is not finite in fp16
inline bool f32_to_f16_bits(float f, uint16_t* out) {
    const __half h = __float2half_rn(f);
    const __half_raw r = static_cast<__half_raw>(h);
    *out = r.x;
    return (r.x & 0x7C00u) != 0x7C00u;
}

namespace ptx {

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
    return ok != 0;
}
// non-blocking probe (try_wait may suspend the thread for a system-dependent time when the phase is not complete)
__device__ __forceinline__ bool mbar_test_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\tmbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
    return ok != 0;
}
// Bounded wait: a protocol bug must trap (and fail the test), never hang the GPU box.  The slow path is kept
// out of line so the ~60 wait sites stay small (the kernel's code footprint matters: one warp per role, nothing
// hides an instruction-cache miss).
static __device__ __noinline__ void mbar_wait_slow(uint32_t bar, uint32_t parity) {
    const long long t0 = clock64();
    while (!mbar_try_wait(bar, parity)) {
        if (clock64() - t0 > 4000000000LL) {
            printf("wm_tc: mbarrier wait timed out (block %d thread %d bar %u parity %u)\n", blockIdx.x, threadIdx.x,
                   bar, parity);
            __trap();
        }
    }
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    if (!mbar_try_wait(bar, parity)) mbar_wait_slow(bar, parity);
}
// the same for a CONVERGED warp whose lanes all wait on the same barrier: the vote makes the branch warp-uniform (no
// reconvergence bookkeeping around the slow path)
// No function call on any path (a call would force the caller's loop state out of the uniform registers): the slow
// path spins in line and traps after ~2 s.
__device__ __forceinline__ void mbar_wait_warp(uint32_t bar, uint32_t parity) {
    if (!__all_sync(0xffffffffu, mbar_try_wait(bar, parity))) {
        const long long t0 = clock64();
        while (!mbar_try_wait(bar, parity))
            if (clock64() - t0 > 4000000000LL) __trap();
    }
}
// Call-free bounded wait for any thread: a function call inside a warpgroup that has raised its register count with
// setmaxnreg keeps ptxas from budgeting that region above the launch-time count (measured: the epilogue of
// wm_tcp_kernel stayed at 128 registers and spilled 4 KB until its waits lost their out-of-line slow path).
__device__ __forceinline__ void mbar_wait_inline(uint32_t bar, uint32_t parity) {
    if (!mbar_try_wait(bar, parity)) {
        const long long t0 = clock64();
        while (!mbar_try_wait(bar, parity))
            if (clock64() - t0 > 4000000000LL) __trap();
    }
}
__device__ __forceinline__ void fence_barrier_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}

__device__ __forceinline__ void tmem_alloc(uint32_t slot_smem, uint32_t ncols) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(slot_smem), "r"(ncols)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t ncols) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}

// D[tmem] (+)= A[smem desc] * B[smem desc]
__device__ __forceinline__ void mma_ss(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t acc) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem),
        "l"(adesc), "l"(bdesc), "r"(idesc), "r"(acc)
        : "memory");
}
// D[tmem] (+)= A[tmem] * B[smem desc]
__device__ __forceinline__ void mma_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t bdesc, uint32_t idesc, uint32_t acc) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}" ::"r"(d_tmem),
        "r"(a_tmem), "l"(bdesc), "r"(idesc), "r"(acc)
        : "memory");
}
__device__ __forceinline__ void mma_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}

__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&r)[32]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
          "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
          "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
          "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
        : "r"(taddr)
        : "memory");
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&r)[16]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
          "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
        : "r"(taddr)
        : "memory");
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_st_wait() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

__device__ __forceinline__ void tmem_st32(uint32_t taddr, const uint32_t (&r)[32]) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], "
        "{%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, "
        "%17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31, %32};" ::"r"(taddr),
        "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]), "r"(r[9]),
        "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]), "r"(r[16]), "r"(r[17]), "r"(r[18]),
        "r"(r[19]), "r"(r[20]), "r"(r[21]), "r"(r[22]), "r"(r[23]), "r"(r[24]), "r"(r[25]), "r"(r[26]), "r"(r[27]),
        "r"(r[28]), "r"(r[29]), "r"(r[30]), "r"(r[31])
        : "memory");
}
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t (&r)[16]) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], "
        "{%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};" ::"r"(taddr),
        "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]), "r"(r[9]),
        "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15])
        : "memory");
}

// Register reallocation between warpgroups (4 consecutive warps; every warp of the group executes the SAME instruction):
// the kernel is compiled for 128 registers per thread, service warps give registers back, register-hungry roles take
// them.  N is a multiple of 8.
template <int N> __device__ __forceinline__ void reg_dealloc() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(N)); }
template <int N> __device__ __forceinline__ void reg_alloc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N)); }

// one lane of a converged warp (always the same one): keeps the MMA operands warp-uniform for the compiler
__device__ __forceinline__ bool elect_one() {
    uint32_t pred;
    asm volatile("{\n\t.reg .pred P;\n\telect.sync _|P, 0xffffffff;\n\tselp.u32 %0, 1, 0, P;\n\t}" : "=r"(pred));
    return pred != 0;
}
__device__ __forceinline__ void named_bar_sync(int id, int nthreads) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// MMA operand pack: two fp32 -> fp16x2 (lo -> bits [0,16), hi -> bits [16,32)), round to nearest, saturating to the
// largest finite fp16 so that an out-of-range activation can never become an infinity inside the recurrence.
// Operand encoding (DESIGN.md §3 S14): the weights are bf16 VALUES; every bf16 value with 2^-14 <= |w| <= 65504 is
// exactly representable in fp16 (11-bit significand vs 8), so the MMAs run kind::f16 on fp16 encodings of the same
// weights (|w| < 2^-14 lands on the fp16 subnormal grid, absolute change <= 3e-8) and the ACTIVATIONS are rounded to
// fp16 (relative 2^-11) instead of bf16 (2^-8): same tensor-pipe rate, 8x less operand rounding noise.
__device__ __forceinline__ uint32_t pack_f16(float lo, float hi) {
    uint32_t r;
    asm("cvt.rn.satfinite.f16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
    return r;
}

// Activations enter the MMAs as fp16 with a SATURATING convert, so a caller-supplied initial latent beyond the fp16 range
// would be silently clamped to 65504: the z_0 loads of the tcgen05 kernels report it (WM_FAULT_RANGE).  Later latents cannot
// leave the range by themselves (LayerNorm / L2 normalisation / the GRU's convex blend bound them by the weights).
__device__ __forceinline__ void range_check(const float4& f, uint32_t* fault) {
    if (fmaxf(fmaxf(fabsf(f.x), fabsf(f.y)), fmaxf(fabsf(f.z), fabsf(f.w))) > 65504.0f) atomicOr(fault, WM_FAULT_RANGE);
}

// GELU, tanh form (hardware tanh.approx): |gelu_tanh - gelu_erf| <= 5e-4 abs, below the bf16 rounding of the
// hidden activations it feeds (DESIGN.md §3 S5).  (A quintic inner polynomial fitted to the erf form, max deviation
// 2.6e-5, was measured: no change in score error, which is dominated by operand rounding, and 4 % slower.)
__device__ __forceinline__ float gelu_fast(float x) {
    const float x2 = x * x;
    const float inner = x * fmaf(0.0356774081f, x2, 0.7978845608f);
    float t;
    asm("tanh.approx.f32 %0, %1;" : "=f"(t) : "f"(inner));
    const float hx = 0.5f * x;
    return fmaf(hx, t, hx);
}

// tanh / logistic sigmoid on the hardware tanh.approx (relative error 2^-11): sigma(x) = 0.5 tanh(0.5 x) + 0.5
__device__ __forceinline__ float tanh_fast(float x) {
    float t;
    asm("tanh.approx.f32 %0, %1;" : "=f"(t) : "f"(x));
    return t;
}
__device__ __forceinline__ float sigmoid_fast(float x) { return fmaf(0.5f, tanh_fast(0.5f * x), 0.5f); }

// Two GELUs at once on the packed fp32x2 pipe (FFMA2/FMUL2/FADD2 halve the epilogue's FP instruction count).
__device__ __forceinline__ uint32_t gelu2_f16(float2 acc, float2 bias) {
    const float2 x = __fadd2_rn(acc, bias);
    const float2 hx = __fmul2_rn(x, make_float2(0.5f, 0.5f));
    const float2 x2 = __fmul2_rn(x, x);
    const float2 pin = __ffma2_rn(x2, make_float2(0.0356774081f, 0.0356774081f), make_float2(0.7978845608f, 0.7978845608f));
    const float2 inner = __fmul2_rn(x, pin);
    float2 t;
    asm("tanh.approx.f32 %0, %1;" : "=f"(t.x) : "f"(inner.x));
    asm("tanh.approx.f32 %0, %1;" : "=f"(t.y) : "f"(inner.y));
    const float2 g = __ffma2_rn(hx, t, hx);
    return pack_f16(g.x, g.y);
}

// Two GELUs (tanh form) entirely on the packed fp16x2 pipe, for accumulators that already carry their bias: one cvt, five
// HMUL2/HFMA2 and ONE MUFU (tanh.approx.f16x2) per pair of elements instead of nine fp32x2 / MUFU instructions.  The
// result is the fp16 MMA operand anyway; the intermediate roundings (2^-11 each) stay below the operand rounding noise
// the tolerance already carries (S5/S14).  Saturating convert: an out-of-range pre-activation becomes 65504,
// never an infinity (gelu(65504) = 65504 in this arithmetic; large negative inputs give exactly 0).
__device__ __forceinline__ uint32_t gelu2_h2(float lo, float hi) {
    const uint32_t x = pack_f16(lo, hi);
    uint32_t x2, pin, inner, t, hx, g;
    asm("mul.f16x2 %0, %1, %1;" : "=r"(x2) : "r"(x));
    asm("fma.rn.f16x2 %0, %1, %2, %3;" : "=r"(pin) : "r"(x2), "r"(0x28912891u), "r"(0x3A623A62u));   // 0.0356774, 0.7978846
    asm("mul.f16x2 %0, %1, %2;" : "=r"(inner) : "r"(x), "r"(pin));
    asm("tanh.approx.f16x2 %0, %1;" : "=r"(t) : "r"(inner));
    asm("mul.f16x2 %0, %1, %2;" : "=r"(hx) : "r"(x), "r"(0x38003800u));                               // 0.5
    asm("fma.rn.f16x2 %0, %1, %2, %1;" : "=r"(g) : "r"(hx), "r"(t));
    return g;
}

// UMMA shared-memory descriptor, K-major, 128B swizzle, 8-row groups 1024 B apart (SBO), version 1 (sm_100).
__device__ __forceinline__ uint64_t smem_desc(uint32_t saddr) {
    const uint32_t lo = ((saddr >> 4) & 0x3FFFu) | (1u << 16);
    const uint32_t hi = (1024u >> 4) | (1u << 14) | (2u << 29);
    return ((uint64_t)hi << 32) | lo;
}
// Same, no swizzle ("interleave"), for a [128 x 16] K-major tile stored as 16-byte rows of 8-row core matrices:
// the two K halves of a core-matrix row group are 128 B apart (LBO), row groups 256 B apart (SBO).
__device__ __forceinline__ uint64_t smem_desc_nosw(uint32_t saddr) {
    const uint32_t lo = ((saddr >> 4) & 0x3FFFu) | ((128u >> 4) << 16);
    const uint32_t hi = (256u >> 4) | (1u << 14);
    return ((uint64_t)hi << 32) | lo;
}
// kind::f16 instruction descriptor: D fp32 (bit 4), A/B fp16 (format fields [7,10) and [10,13) = 0; 1 would be bf16),
// both K-major, M = 128, N = 128.
constexpr uint32_t IDESC = (1u << 4) | ((128u >> 3) << 17) | ((128u >> 4) << 24);
// the same with N = 256 (one MMA = 128 tensor cycles: half the issue work per FLOP of N = 128)
constexpr uint32_t IDESC_N256 = (1u << 4) | ((256u >> 3) << 17) | ((128u >> 4) << 24);

// ------------------------------------------------------------------------------------------------ tile helpers
__device__ __forceinline__ int find_seg(const int32_t* __restrict__ off, int S, int cand) {
    int lo = 0, hi = S;
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (__ldg(off + mid) <= cand) lo = mid; else hi = mid;
    }
    return lo;
}

// Row metadata of sorted position i (tile * rows_per_tile + row): candidate index (-1 = dead row), clamped length, subgraph (z0 / hw row).
__device__ __forceinline__ void row_meta(const CallArgs& a, int64_t i, int& cand, int& len, int& seg, bool report) {
    cand = -1; len = 0; seg = 0;
    if (i < a.B) {
        cand = a.perm ? __ldg(a.perm + i) : (int)i;
        len = __ldg(a.lengths + cand);
        if (len < 0 || len > a.T_max) {
            if (report) atomicOr(a.fault, WM_FAULT_LEN);
            len = len < 0 ? 0 : a.T_max;
        }
        seg = a.offsets ? find_seg(a.offsets, a.S, cand) : cand;
    }
}

// Prefix-latent reuse (wm_rollout_score_from): first position the rollout applies for this candidate; 0 otherwise.
__device__ __forceinline__ int row_start(const CallArgs& a, int cand, int len) {
    return (a.start && cand >= 0) ? clamp_start(__ldg(a.start + cand), len) : 0;
}

// Row of init_states that holds candidate `cand`'s initial latent: its subgraph's (seg), or the banked row
// init_index names (clamped into [0, n_init), WM_FAULT_INDEX raised when it was outside).
__device__ __forceinline__ size_t row_init(const CallArgs& a, int cand, int seg) {
    if (!a.init_index || cand < 0) return (size_t)seg;
    long long i = __ldg(a.init_index + cand);
    if (i < 0 || i >= a.n_init) {
        atomicOr(a.fault, WM_FAULT_INDEX);
        i = i < 0 ? 0 : a.n_init - 1;
    }
    return (size_t)i;
}

// byte offset of the 16-byte chunk `chunk` (8 bf16 columns) of row `row` inside a SW128 K-major K-block tile
__device__ __forceinline__ uint32_t sw128_off(int row, int chunk) {
    return (uint32_t)row * 128u + (uint32_t)((chunk ^ (row & 7)) << 4);
}


// ------------------------------------------------------------------------------------------------ CTA pair (cta_group::2)
__device__ __forceinline__ uint32_t cluster_ctarank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// shared::cluster address of `saddr` (a shared::cta address of this CTA) in CTA `rank` of the cluster
__device__ __forceinline__ uint32_t mapa(uint32_t saddr, uint32_t rank) {
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(saddr), "r"(rank));
    return r;
}
// arrive on a barrier anywhere in the cluster (address from mapa), release at cluster scope
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t cluster_addr) {
    asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}
// The same with the default semantics (release at CTA scope), as CUTLASS's ClusterBarrier::arrive(cta_id) does.  The
// cluster-scope release above compiles to MEMBAR.ALL.GPU + ERRBAR + CGAERRBAR in front of the arrive: measured ~1500
// cycles per publish in wm_tcp_kernel (more than the GELU it publishes).  What the pair kernels hand over is either
// tensor memory (completed by tcgen05.wait::st and ordered by tcgen05.fence::before_thread_sync) or the arriving CTA's
// OWN shared memory, made visible to its own async proxy by fence.proxy.async before the arrive; the MMA the leader
// then issues reads each CTA's operands through that CTA's own SM, so no generic-proxy data crosses CTAs.
__device__ __forceinline__ void mbar_arrive_remote(uint32_t cluster_addr) {
    asm volatile("mbarrier.arrive.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait_cluster(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
    return ok != 0;
}
static __device__ __noinline__ void mbar_wait_cluster_slow(uint32_t bar, uint32_t parity) {
    const long long t0 = clock64();
    while (!mbar_try_wait_cluster(bar, parity)) {
        if (clock64() - t0 > 4000000000LL) {
            printf("wm_tc2: cluster mbarrier wait timed out (block %d thread %d bar %u parity %u)\n", blockIdx.x,
                   threadIdx.x, bar, parity);
            __trap();
        }
    }
}
// wait on a LOCAL barrier whose arrivals come from both CTAs of the pair
__device__ __forceinline__ void mbar_wait_cluster(uint32_t bar, uint32_t parity) {
    if (!mbar_try_wait_cluster(bar, parity)) mbar_wait_cluster_slow(bar, parity);
}
__device__ __forceinline__ void mbar_wait_cluster_warp(uint32_t bar, uint32_t parity) {
    if (!__all_sync(0xffffffffu, mbar_try_wait_cluster(bar, parity))) {
        const long long t0 = clock64();
        while (!mbar_try_wait_cluster(bar, parity))
            if (clock64() - t0 > 4000000000LL) __trap();
    }
}
// One warp of EACH CTA of the pair (same warp id) allocates / frees; both get the same column base.
__device__ __forceinline__ void tmem_alloc2(uint32_t slot_smem, uint32_t ncols) {
    asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(slot_smem), "r"(ncols)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc2(uint32_t taddr, uint32_t ncols) {
    asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}
// Pair MMA, issued by the leader CTA only: D (+)= A * B with M = 128 (64 rows per CTA), B split by N halves.
// The descriptors are CTA-relative shared-memory offsets, valid in both CTAs.
__device__ __forceinline__ void mma_ss2(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t acc) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem),
        "l"(adesc), "l"(bdesc), "r"(idesc), "r"(acc)
        : "memory");
}
// completion of all prior pair MMAs -> arrive on the barrier at this offset in BOTH CTAs
__device__ __forceinline__ void mma_commit2(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(bar),
                 "h"((uint16_t)3)
                 : "memory");
}
// TMA tile load into THIS CTA's shared memory whose complete_tx lands on the LEADER CTA's barrier (peer bit cleared)
__device__ __forceinline__ void tma_load_2sm(uint32_t dst, const void* tmap, int x, int y, uint32_t bar) {
    asm volatile(
        "cp.async.bulk.tensor.2d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];" ::"r"(dst),
        "l"(tmap), "r"(bar & 0xFEFFFFFFu), "r"(x), "r"(y)
        : "memory");
}
// low word of the SW128 K-major descriptor of a tile at shared address saddr (the high word is DESC_HI for every
// tile); a tile `bytes` further on has low word + (bytes >> 4), the next K = 16 step inside a tile + 2
constexpr uint32_t DESC_HI = (1024u >> 4) | (1u << 14) | (2u << 29);
__device__ __forceinline__ uint32_t smem_desc_lo(uint32_t saddr) { return ((saddr >> 4) & 0x3FFFu) | (1u << 16); }
__device__ __forceinline__ uint64_t desc_of(uint32_t lo) { return ((uint64_t)DESC_HI << 32) | lo; }

// kind::f16 instruction descriptor of the pair MMA: D fp32, A/B fp16, both K-major, M = 128, N = 256
constexpr uint32_t idesc_pair(uint32_t n) { return (1u << 4) | ((n >> 3) << 17) | ((128u >> 4) << 24); }
constexpr uint32_t IDESC2 = idesc_pair(256);

}  // namespace ptx
}  // namespace wm
