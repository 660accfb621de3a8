// hb_tc_common.cuh -- shared by the tensor-core surrogate kernels (hb_sur_tc.cu: weights resident in shared
// memory; hb_sur_tcs.cu: weights streamed from L2): tile constants, PTX wrappers (mbarrier, bulk copy, tcgen05
// alloc / mma / commit / ld, descriptors), the hidden-layer epilogue step.
#pragma once
#include "hb_device.cuh"

#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cstdio>
#include <cstdlib>
#include <cstring>

namespace {

constexpr int TILE_M = 128;
constexpr int A_SLAB_BYTES = TILE_M * 128;       // 128 rows x 64 16-bit elements, 128-byte swizzle
constexpr int A0_BYTES = TILE_M * 32;            // layer-0 operand: 128 rows x 16 elements, no swizzle
constexpr int IO_WARP0 = 0;                      // warps 0..3
constexpr int EPI_WARP0 = 4;                     // warps 4..4+4G-1; then the producer warp, then the MMA warp
constexpr int tc_threads(int g) { return 32 * (EPI_WARP0 + 4 * g + 2); }
constexpr int IN_STAGES = 2;
constexpr int STAGE_BYTES = 6 * TILE_M * 4;
constexpr int MAX_SLABS = 4;                     // hidden width <= 256
constexpr size_t SMEM_LIMIT = 227 * 1024;

// ------------------------------------------------------------------------------- PTX wrappers
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive_local(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
// arrive on the barrier at the same offset in CTA `rank` of the cluster (rank 0 = MMA leader).  No
// .release.cluster qualifier: that form costs a MEMBAR.ALL.GPU per arrive (measured, profiles/); the data the
// arrive publishes is shared memory already made visible to the async proxy by fence.proxy.async.
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t bar, uint32_t rank) {
    uint32_t remote;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(remote) : "r"(bar), "r"(rank));
    asm volatile("mbarrier.arrive.shared::cluster.b64 _, [%0];" ::"r"(remote) : "memory");
}
// non-blocking probe (try_wait may suspend the thread for a while when the phase is still open)
__device__ __forceinline__ uint32_t mbar_test(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
                 "selp.u32 %0, 1, 0, p;\n\t}" : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok;
}
__device__ __forceinline__ uint32_t mbar_try(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
                 "selp.u32 %0, 1, 0, p;\n\t}" : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok;
}
// try_wait with a suspend-time hint: the thread sleeps in hardware until the phase completes (or the hint
// expires) instead of spinning through the issue slots of the warps that do the work
__device__ __forceinline__ uint32_t mbar_try_sleep(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\t"
                 "selp.u32 %0, 1, 0, p;\n\t}" : "=r"(ok) : "r"(bar), "r"(parity), "r"(200000u) : "memory");
    return ok;
}
// Guarded wait of every warp role but the MMA issuer.  FAST: latency-critical waiters poll with the plain try_wait (it
// suspends the thread for a short, bounded time and wakes it when the phase completes); the others pass a long
// suspend-time hint, which costs less issue bandwidth and wakes later.  The hang guard (~2 s: a protocol bug must not
// hang the GPU) is a bare trap: a printf in the waiting loop -- or a call to a function that holds it -- cost every wait
// 100 cycles more even when the phase had completed long ago (152 against 55 cycles, csrc/microbench/hb_epi_cost.cu),
// and, worse, made ptxas give up the uniform datapath in whatever code surrounds the wait (see mbar_spin).
template <bool FAST>
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    if (mbar_try(bar, parity)) return;
    const long long t0 = clock64();
    while (!(FAST ? mbar_try(bar, parity) : mbar_try_sleep(bar, parity))) {
        if (clock64() - t0 > 4000000000LL) __trap();
    }
}
// Wait of the MMA-issuing warp: a bare spin on test_wait, no guard.
// Why bare.  The issuing warp walks its schedule in warp-uniform control flow and feeds tcgen05.mma from UNIFORM
// registers (descriptors, tensor-memory addresses).  ptxas keeps that arithmetic on the uniform datapath only while it can
// prove the warp converged; a trap, a printf or a call inside a wait loop of that region makes it fall back to
// per-thread registers plus an R2UR (and R2UR.BROADCAST / WARPSYNC) in front of every MMA: 278 R2UR instead of 34 in the
// issuing region of hb_sur_tc2_kernel, 2.21 ms instead of 2.05 ms on C3 (profiles/r2_issuer_codegen.md).
// Why that is safe.  Every wait of an issuer precedes MMAs and a tcgen05.commit that guarded waiters (epilogue and IO
// warps, mbar_wait above) depend on: an issuer stuck here surfaces as THEIR timeout, and the trap ends the whole grid.
__device__ __forceinline__ void mbar_spin(uint32_t bar, uint32_t parity) {
    while (!mbar_test(bar, parity)) {}
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

template <int CG>
__device__ __forceinline__ void tmem_alloc(uint32_t dst_smem, uint32_t cols) {
    if (CG == 1) asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(dst_smem), "r"(cols) : "memory");
    else asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(dst_smem), "r"(cols) : "memory");
}
template <int CG>
__device__ __forceinline__ void tmem_relinquish() {
    if (CG == 1) asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    else asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
}
template <int CG>
__device__ __forceinline__ void tmem_dealloc(uint32_t addr, uint32_t cols) {
    if (CG == 1) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(addr), "r"(cols) : "memory");
    else asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(addr), "r"(cols) : "memory");
}
// D[tmem] (+)= A[smem desc] * B[smem desc];  T32: kind::tf32 (32-bit operands, K = 8), else kind::f16 (K = 16)
template <int CG, bool ACC, bool T32 = false>
__device__ __forceinline__ void umma(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc) {
    if (CG == 1 && !T32)
        asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                     "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
                     ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "n"(ACC ? 1 : 0) : "memory");
    else if (!T32)
        asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                     "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n\t}"
                     ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "n"(ACC ? 1 : 0) : "memory");
    else if (CG == 1)
        asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                     "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}"
                     ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "n"(ACC ? 1 : 0) : "memory");
    else
        asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                     "tcgen05.mma.cta_group::2.kind::tf32 [%0], %1, %2, %3, p;\n\t}"
                     ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "n"(ACC ? 1 : 0) : "memory");
}
__device__ __forceinline__ bool elect_one() {
    uint32_t pred;
    asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(pred));
    return pred != 0;
}
// all MMAs issued so far by this thread arrive on `bar` (in both CTAs of a pair) when they complete
template <int CG>
__device__ __forceinline__ void umma_commit(uint32_t bar) {
    if (CG == 1)
        asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
    else
        asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;"
                     ::"r"(bar), "h"((uint16_t)3) : "memory");
}
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&r)[32]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,"
        "%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
          "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]),
          "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]),
          "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
        : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_ld8(uint32_t taddr, uint32_t (&r)[8]) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
                 : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

__device__ __forceinline__ uint32_t cluster_rank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}

// K-major, 128-byte swizzle shared-memory matrix descriptor (sm_100): start address, LBO = 1 (unused for
// swizzled K-major), SBO = 1024 B between 8-row groups, version 1, layout type 2 (SWIZZLE_128B).
__device__ __forceinline__ uint64_t make_desc(uint32_t saddr) {
    uint64_t d = (uint64_t)((saddr & 0x3FFFFu) >> 4);
    d |= (uint64_t)1 << 16;
    d |= (uint64_t)(1024 >> 4) << 32;
    d |= (uint64_t)1 << 46;
    d |= (uint64_t)2 << 61;
    return d;
}

template <bool F16>
__device__ __forceinline__ uint32_t pack2(float lo, float hi) {   // element at the lower address = lo
    uint32_t d;
    if (F16) asm("cvt.rn.f16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(hi), "f"(lo));
    else asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(hi), "f"(lo));
    return d;
}
template <bool F16>
__device__ __forceinline__ float round16(float v) {   // value after rounding to the operand type
    if (F16) return __half2float(__float2half_rn(v));
    return __bfloat162float(__float2bfloat16_rn(v));
}


__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&r)[16]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
          "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
        : "r"(taddr) : "memory");
}
template <int CW>
__device__ __forceinline__ void tmem_ld(uint32_t taddr, uint32_t (&r)[CW]) {
    static_assert(CW == 16 || CW == 32, "column chunk");
    if constexpr (CW == 32) tmem_ld32(taddr, r);
    else tmem_ld16(taddr, r);
}

// D[tmem] (+)= A[tmem] * B[smem]: the A operand is read from tensor memory (lane = row, one 32-bit column = two
// consecutive K elements, so one K = 16 step is 8 columns); 16-bit kinds only.
template <int CG, bool ACC>
__device__ __forceinline__ void umma_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc) {
    if (CG == 1)
        asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                     "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}"
                     ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(idesc), "n"(ACC ? 1 : 0) : "memory");
    else
        asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                     "tcgen05.mma.cta_group::2.kind::f16 [%0], [%1], %2, %3, p;\n\t}"
                     ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(idesc), "n"(ACC ? 1 : 0) : "memory");
}
// 16 columns of this thread's TMEM lane <- registers
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t (&r)[16]) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};"
        ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]),
          "r"(r[8]), "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]) : "memory");
}
__device__ __forceinline__ void tmem_st_wait() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
// K-major, no swizzle (layer 0, K = 16): core matrices of 8 rows x 16 bytes; the two K chunks of an 8-row
// group sit 128 B apart (LBO), 8-row groups 256 B apart (SBO).
__device__ __forceinline__ uint64_t make_desc_l0(uint32_t saddr) {
    uint64_t d = (uint64_t)((saddr & 0x3FFFFu) >> 4);
    d |= (uint64_t)(128 >> 4) << 16;
    d |= (uint64_t)(256 >> 4) << 32;
    d |= (uint64_t)1 << 46;
    return d;
}

// (a + bias) for two adjacent accumulator columns in one FADD2
__device__ __forceinline__ void add2(float& a0, float& a1, float b0, float b1) {
    uint64_t A, B;
    asm("mov.b64 %0, {%1, %2};" : "=l"(A) : "f"(a0), "f"(a1));
    asm("mov.b64 %0, {%1, %2};" : "=l"(B) : "f"(b0), "f"(b1));
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(A) : "l"(A), "l"(B));
    asm("mov.b64 {%0, %1}, %2;" : "=f"(a0), "=f"(a1) : "l"(A));
}
template <bool F16>
__device__ __forceinline__ uint32_t pack2_relu(float lo, float hi) {   // max(.,0) fused into the conversion
    uint32_t d;
    if (F16) asm("cvt.rn.relu.f16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(hi), "f"(lo));
    else asm("cvt.rn.relu.bf16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(hi), "f"(lo));
    return d;
}
// sigma(z0 + b0), sigma(z1 + b1) -> two packed 16-bit operands (Eq. 1, Eq. 2, tanh)
template <int ACT, bool F16>
__device__ __forceinline__ uint32_t act_pack(float z0, float z1, float slope) {
    if (ACT == 1) return pack2_relu<F16>(z0, z1);
    if (ACT == 2) { z0 = z0 >= 0.0f ? z0 : slope * z0; z1 = z1 >= 0.0f ? z1 : slope * z1; }
    if (ACT == 3) { z0 = hb_tanh_approx(z0); z1 = hb_tanh_approx(z1); }
    return pack2<F16>(z0, z1);
}

// One hidden-layer epilogue step of one warp: CW accumulator columns [c0, c0+CW) of its 32 lanes -> bias,
// sigma, 16-bit, stored as CW/8 16-byte chunks of the next A operand (row = lane's particle).
template <int CW, int ACT, bool F16>
__device__ __forceinline__ void epi_store(const uint32_t (&r)[CW], const float* __restrict__ bl, int c0, float slope,
                                          uint32_t a_row, uint32_t sw) {
    uint32_t q[CW / 2];
#pragma unroll
    for (int k = 0; k < CW / 4; ++k) {
        const float4 b4 = *reinterpret_cast<const float4*>(bl + c0 + 4 * k);
        float v0 = __uint_as_float(r[4 * k]), v1 = __uint_as_float(r[4 * k + 1]);
        float v2 = __uint_as_float(r[4 * k + 2]), v3 = __uint_as_float(r[4 * k + 3]);
        add2(v0, v1, b4.x, b4.y);
        add2(v2, v3, b4.z, b4.w);
        q[2 * k] = act_pack<ACT, F16>(v0, v1, slope);
        q[2 * k + 1] = act_pack<ACT, F16>(v2, v3, slope);
    }
    const uint32_t slab = a_row + (uint32_t)(c0 >> 6) * A_SLAB_BYTES;
    const uint32_t ch0 = (uint32_t)((c0 & 63) >> 3);
#pragma unroll
    for (int k = 0; k < CW / 8; ++k)
        asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(slab + (((ch0 + k) ^ sw) << 4)),
                     "r"(q[4 * k]), "r"(q[4 * k + 1]), "r"(q[4 * k + 2]), "r"(q[4 * k + 3]) : "memory");
}


// As epi_store without the bias: the accumulator already holds W a + b (the bias went in as an MMA of its own).
template <int CW, int ACT, bool F16>
__device__ __forceinline__ void epi_store_nb(const uint32_t (&r)[CW], int c0, float slope, uint32_t a_row, uint32_t sw) {
    uint32_t q[CW / 2];
#pragma unroll
    for (int k = 0; k < CW / 2; ++k)
        q[k] = act_pack<ACT, F16>(__uint_as_float(r[2 * k]), __uint_as_float(r[2 * k + 1]), slope);
    const uint32_t slab = a_row + (uint32_t)(c0 >> 6) * A_SLAB_BYTES;
    const uint32_t ch0 = (uint32_t)((c0 & 63) >> 3);
#pragma unroll
    for (int k = 0; k < CW / 8; ++k)
        asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(slab + (((ch0 + k) ^ sw) << 4)),
                     "r"(q[4 * k]), "r"(q[4 * k + 1]), "r"(q[4 * k + 2]), "r"(q[4 * k + 3]) : "memory");
}

// One hidden-layer epilogue step of one warp with the next operand kept in tensor memory: 32 accumulator columns
// (bias already inside) -> sigma, round to 16 bit -> 16 packed columns, written over the first half of the very
// columns they came from (taddr = lane | first column of the chunk).
template <int ACT, bool F16>
__device__ __forceinline__ void epi_store_tmem(const uint32_t (&r)[32], uint32_t taddr, float slope) {
    uint32_t q[16];
#pragma unroll
    for (int k = 0; k < 16; ++k)
        q[k] = act_pack<ACT, F16>(__uint_as_float(r[2 * k]), __uint_as_float(r[2 * k + 1]), slope);
    tmem_st16(taddr, q);
}

// a4: six s-coordinates of one particle -> the K = 16 layer-0 operand row  hi0..hi5, lo0..lo5, 0, 0, 0, 0
// (hi = value rounded to the operand type, lo = rounded remainder), as two 16-byte chunks.
template <bool F16>
__device__ __forceinline__ void tc_make_a0_row(const HbSurDev& sd, bool valid, const float (&c)[6], uint32_t (&q0)[4],
                                               uint32_t (&q1)[4]) {
    float nin[6] = {0, 0, 0, 0, 0, 0};
    if (valid) hb_sur_prologue(sd, c[0], c[1], c[2], c[3], c[4], c[5], nin);
    float lo[6];
#pragma unroll
    for (int j = 0; j < 6; ++j) lo[j] = nin[j] - round16<F16>(nin[j]);
    q0[0] = pack2<F16>(nin[0], nin[1]); q0[1] = pack2<F16>(nin[2], nin[3]); q0[2] = pack2<F16>(nin[4], nin[5]);
    q0[3] = pack2<F16>(lo[0], lo[1]);
    q1[0] = pack2<F16>(lo[2], lo[3]); q1[1] = pack2<F16>(lo[4], lo[5]); q1[2] = 0u; q1[3] = 0u;
}
__device__ __forceinline__ void sts128(uint32_t addr, const uint32_t (&q)[4]) {
    asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(addr), "r"(q[0]), "r"(q[1]), "r"(q[2]), "r"(q[3]) : "memory");
}

// Same step, but into one given 16 KB slab (ring slot): `slab_row` = address of this thread's row in the slab,
// `ch0` = first 16-byte chunk of the row the CW columns go to, `bl` already points at the first column's bias.
template <int CW, int ACT, bool F16>
__device__ __forceinline__ void epi_store_slab(const uint32_t (&r)[CW], const float* __restrict__ bl, uint32_t ch0,
                                               float slope, uint32_t slab_row, uint32_t sw) {
    uint32_t q[CW / 2];
#pragma unroll
    for (int k = 0; k < CW / 4; ++k) {
        const float4 b4 = *reinterpret_cast<const float4*>(bl + 4 * k);
        float v0 = __uint_as_float(r[4 * k]), v1 = __uint_as_float(r[4 * k + 1]);
        float v2 = __uint_as_float(r[4 * k + 2]), v3 = __uint_as_float(r[4 * k + 3]);
        add2(v0, v1, b4.x, b4.y);
        add2(v2, v3, b4.z, b4.w);
        q[2 * k] = act_pack<ACT, F16>(v0, v1, slope);
        q[2 * k + 1] = act_pack<ACT, F16>(v2, v3, slope);
    }
#pragma unroll
    for (int k = 0; k < CW / 8; ++k)
        asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(slab_row + (((ch0 + k) ^ sw) << 4)),
                     "r"(q[4 * k]), "r"(q[4 * k + 1]), "r"(q[4 * k + 2]), "r"(q[4 * k + 3]) : "memory");
}

// ---- tf32 operands (HB_PREC_TF32): 32-bit elements, 32 per 128-byte slab row, K = 8 per MMA
__device__ __forceinline__ float to_tf32(float v) {           // round to nearest (ties away), low 13 bits zero
    uint32_t d;
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(d) : "f"(v));
    return __uint_as_float(d);
}
// K-major, no swizzle, 32-bit elements, K = 16 (layer 0): core matrices of 8 rows x 16 bytes (4 elements); the four
// K chunks of an 8-row group sit 128 B apart (LBO), 8-row groups 512 B apart (SBO).
__device__ __forceinline__ uint64_t make_desc_l0_t32(uint32_t saddr) {
    uint64_t d = (uint64_t)((saddr & 0x3FFFFu) >> 4);
    d |= (uint64_t)(128 >> 4) << 16;
    d |= (uint64_t)(512 >> 4) << 32;
    d |= (uint64_t)1 << 46;
    return d;
}
// One hidden-layer epilogue step of one warp for tf32: 32 accumulator columns -> bias, sigma, tf32, one full
// 128-byte slab row (eight 16-byte chunks, swizzled).
template <int ACT>
__device__ __forceinline__ void epi_store_t32(const uint32_t (&r)[32], const float* __restrict__ bl, float slope,
                                              uint32_t slab_row, uint32_t sw) {
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        const float4 b4 = *reinterpret_cast<const float4*>(bl + 4 * k);
        float v[4] = {__uint_as_float(r[4 * k]) + b4.x, __uint_as_float(r[4 * k + 1]) + b4.y,
                      __uint_as_float(r[4 * k + 2]) + b4.z, __uint_as_float(r[4 * k + 3]) + b4.w};
        uint32_t q[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) q[e] = __float_as_uint(to_tf32(hb_activate<ACT, true>(v[e], slope)));
        asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(slab_row + ((((uint32_t)k) ^ sw) << 4)),
                     "r"(q[0]), "r"(q[1]), "r"(q[2]), "r"(q[3]) : "memory");
    }
}
// a4 for tf32: the K = 16 layer-0 operand row  hi0..hi5, lo0..lo5, 0, 0, 0, 0  as four 16-byte chunks
__device__ __forceinline__ void tc_make_a0_row_t32(const HbSurDev& sd, bool valid, const float (&c)[6], uint32_t (&q)[4][4]) {
    float nin[6] = {0, 0, 0, 0, 0, 0};
    if (valid) hb_sur_prologue(sd, c[0], c[1], c[2], c[3], c[4], c[5], nin);
    float e[16];
#pragma unroll
    for (int j = 0; j < 6; ++j) { e[j] = to_tf32(nin[j]); e[6 + j] = to_tf32(nin[j] - e[j]); }
    e[12] = e[13] = e[14] = e[15] = 0.0f;
#pragma unroll
    for (int k = 0; k < 4; ++k)
#pragma unroll
        for (int i = 0; i < 4; ++i) q[k][i] = __float_as_uint(e[4 * k + i]);
}

}  // namespace
