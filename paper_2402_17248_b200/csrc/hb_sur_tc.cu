// hb_sur_tc.cu -- surrogate stage on the 5th-gen tensor cores (HB_PREC_BF16 / HB_PREC_F16): rows a4-a6.
//
// Per 128-particle tile (one TMEM lane per particle):
//   a4  bulk-async copies (TMA engine, cp.async.bulk + mbarrier complete_tx) stage the six coordinate
//       rows of the tile in shared memory; worker threads convert s->t (R6, deviation form), normalise
//       (R8), split each input into hi + lo 16-bit parts (K padded 6 -> 16) and write the A operand.
//   a5  one elected thread issues tcgen05.mma (kind::f16, fp32 accumulate in TMEM) for L_0 .. L_l (Eq. 3);
//       between layers the worker warps read the accumulator with tcgen05.ld, add the bias in fp32,
//       apply sigma (Eq. 1/2 or tanh), round to 16 bit and write the next A operand straight into the
//       128-byte-swizzled K-major shared-memory layout the MMA reads.  Hidden activations never leave
//       the SM.
//   a6  the last accumulator (6 of 16 columns) is de-normalised (R8), moved to the new reference and
//       converted t->s (R6, R7), stored coalesced, and folded into the fp64 moment sums (R10).
// Weights are packed on the host into the exact shared-memory image (hb_tc_pack_weights) and stay
// resident in shared memory for the whole kernel.  CG = 2 pairs two SMs (cta_group::2, M = 256): each
// CTA holds half of every weight matrix (N split), which is what lets 6-256^3-6 stay resident.
#include "hb_device.cuh"

#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cstdio>
#include <cstdlib>
#include <cstring>

namespace {

constexpr int TILE_M = 128;
constexpr int A_SLAB_BYTES = TILE_M * 128;       // 128 rows x 64 16-bit elements
constexpr int WORKER_WARPS = 8;                  // two warps per TMEM lane quarter (column halves)
constexpr int THREADS = 64 + 32 * WORKER_WARPS;  // warp 0: copy producer, warp 1: MMA issuer
constexpr int IN_STAGES = 2;
constexpr int STAGE_BYTES = 6 * TILE_M * 4;
constexpr size_t SMEM_LIMIT = 227 * 1024;

struct TcPlan {
    int n_linear;
    int ksteps[HB_MAX_LINEAR];        // K = 16 MMA steps of layer l
    int nslab[HB_MAX_LINEAR];         // 64-wide K slabs of layer l's operands
    int npad[HB_MAX_LINEAR];          // padded fan-out (whole layer, both CTAs of a pair)
    int w_off[HB_MAX_LINEAR];         // smem byte offset of layer l's weight slabs (this CTA's rows)
    int w_slab_bytes[HB_MAX_LINEAR];  // (npad / CG) * 128
    int bias_off[HB_MAX_LINEAR];      // float offset inside the smem bias block
    int a_off, stage_off, bias_base, bar_off, red_off, total;
    int tmem_cols;
    int w_bytes_total;                // bytes this CTA loads
};

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
// arrive on the barrier at the same offset in CTA `rank` of the cluster (rank 0 = MMA leader)
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t bar, uint32_t rank) {
    uint32_t remote;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(remote) : "r"(bar), "r"(rank));
    asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(remote) : "memory");
}
template <bool CLUSTER_SCOPE>
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok = 0;
    const long long t0 = clock64();
    while (true) {
        if (CLUSTER_SCOPE)
            asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%1], %2;\n\t"
                         "selp.u32 %0, 1, 0, p;\n\t}" : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
        else
            asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
                         "selp.u32 %0, 1, 0, p;\n\t}" : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
        if (ok) break;
        if (clock64() - t0 > 4000000000LL) {   // ~2 s: a protocol bug must not hang the GPU
            printf("hb_sur_tc: mbarrier timeout (block %d thread %d bar %u parity %u)\n", blockIdx.x, threadIdx.x, bar, parity);
            __trap();
        }
    }
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
// D[tmem] (+)= A[smem desc] * B[smem desc]
template <int CG>
__device__ __forceinline__ void umma(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
    if (CG == 1)
        asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                     "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
                     ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate) : "memory");
    else
        asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                     "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n\t}"
                     ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate) : "memory");
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

// ------------------------------------------------------------------------------- kernel
template <int CG, int ACT, bool F16>
__global__ void __launch_bounds__(THREADS, 1)
hb_sur_tc_kernel(HbParticles p, size_t n, const __grid_constant__ HbSurDev sd, const __grid_constant__ TcPlan pl,
                 double* __restrict__ partials) {
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    // the 128-byte swizzle atoms (8 rows x 128 B) must sit on 1024-byte boundaries of the shared window
    unsigned char* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    const uint32_t sbase = smem_u32(smem);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const uint32_t rank = CG == 1 ? 0u : cluster_rank();
    const size_t ntiles = (n + TILE_M - 1) / TILE_M;
    const size_t ngroups = (ntiles + CG - 1) / CG;
    const size_t cluster_id = blockIdx.x / CG, nclusters = gridDim.x / CG;

    // barriers: [0] w_full, [1..2] in_full, [3..4] in_empty, [5] a_ready, [6] d_full; then the TMEM pointer
    const uint32_t bar0 = sbase + pl.bar_off;
    const uint32_t bar_w = bar0, bar_in_full = bar0 + 8, bar_in_empty = bar0 + 24, bar_a = bar0 + 40, bar_d = bar0 + 48;
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + pl.bar_off + 64);
    float* bias_s = reinterpret_cast<float*>(smem + pl.bias_base);

    if (tid == 0) {
        mbar_init(bar_w, 1);
        for (int s = 0; s < IN_STAGES; ++s) { mbar_init(bar_in_full + 8 * s, 1); mbar_init(bar_in_empty + 8 * s, 4); }
        mbar_init(bar_a, WORKER_WARPS * CG);
        mbar_init(bar_d, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 1) {
        tmem_alloc<CG>(smem_u32(tmem_slot), (uint32_t)pl.tmem_cols);
        tmem_relinquish<CG>();
    }
    // biases -> shared (all layers)
    {
        int total = 0;
        for (int l = 0; l < pl.n_linear; ++l) total = pl.bias_off[l] + pl.npad[l];
        for (int i = tid; i < total; i += THREADS) {
            int l = 0;
            while (l + 1 < pl.n_linear && i >= pl.bias_off[l + 1]) ++l;
            bias_s[i] = sd.btc[sd.btc_off[l] + (i - pl.bias_off[l])];
        }
    }
    tc_fence_before();
    __syncthreads();
    if (CG == 2) cluster_sync_all();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    if (warp == 0) {
        // ===================================================== producer: weights once, then particle tiles
        if (lane == 0) {
            mbar_expect_tx(bar_w, (uint32_t)pl.w_bytes_total);
            const unsigned char* wg = reinterpret_cast<const unsigned char*>(sd.wtc);
            for (int l = 0; l < pl.n_linear; ++l)
                for (int s = 0; s < pl.nslab[l]; ++s) {
                    const unsigned char* src = wg + sd.wtc_off[l] + (size_t)s * pl.npad[l] * 128 + (size_t)rank * pl.w_slab_bytes[l];
                    bulk_g2s(sbase + pl.w_off[l] + s * pl.w_slab_bytes[l], src, (uint32_t)pl.w_slab_bytes[l], bar_w);
                }
            int stage = 0;
            uint32_t ph = 0;
            for (size_t g = cluster_id; g < ngroups; g += nclusters) {
                const size_t tile = g * CG + rank;
                const bool full = tile < ntiles && (tile + 1) * TILE_M <= n;
                if (full) {
                    mbar_wait<false>(bar_in_empty + 8 * stage, ph ^ 1);
                    mbar_expect_tx(bar_in_full + 8 * stage, STAGE_BYTES);
                    for (int j = 0; j < 6; ++j)
                        bulk_g2s(sbase + pl.stage_off + stage * STAGE_BYTES + j * TILE_M * 4, p.v[j] + tile * TILE_M,
                                 TILE_M * 4, bar_in_full + 8 * stage);
                    stage ^= 1;
                    if (stage == 0) ph ^= 1;
                }
            }
        }
        __syncwarp();
    } else if (warp == 1) {
        // ===================================================== MMA issuer (leader CTA of the pair only)
        if (rank == 0 && lane == 0) {
            const uint32_t fmt = F16 ? 0u : 1u;
            const uint32_t idesc_base = (1u << 4) | (fmt << 7) | (fmt << 10) | ((uint32_t)((TILE_M * CG) >> 4) << 24);
            uint32_t pa = 0;
            for (size_t g = cluster_id; g < ngroups; g += nclusters) {
                for (int l = 0; l < pl.n_linear; ++l) {
                    mbar_wait<CG == 2>(bar_a, pa);
                    pa ^= 1;
                    tc_fence_after();
                    const int npad = pl.npad[l];
                    for (int n0 = 0; n0 < npad; n0 += 256) {
                        const int nb = min(256, npad - n0);
                        const uint32_t idesc = idesc_base | ((uint32_t)(nb >> 3) << 17);
                        const uint32_t b_row0 = sbase + pl.w_off[l] + (n0 / CG) * 128;
                        for (int ks = 0; ks < pl.ksteps[l]; ++ks) {
                            const uint64_t ad = make_desc(sbase + pl.a_off + (ks >> 2) * A_SLAB_BYTES + (ks & 3) * 32);
                            const uint64_t bd = make_desc(b_row0 + (ks >> 2) * pl.w_slab_bytes[l] + (ks & 3) * 32);
                            umma<CG>(tmem_base + n0, ad, bd, idesc, ks > 0 ? 1u : 0u);
                        }
                    }
                    umma_commit<CG>(bar_d);
                }
            }
        }
        __syncwarp();
    } else {
        // ===================================================== workers: prologue, layer epilogues, output
        const int wq = warp & 3;                 // TMEM lane quarter this warp may access
        const int half = (warp - 2) >> 2;        // column half
        const int row = 32 * wq + lane;          // tile row = TMEM lane = particle within the tile
        const uint32_t a_row = sbase + pl.a_off + row * 128;
        const uint32_t sw = (uint32_t)(row & 7);
        const uint32_t tlane = tmem_base + ((uint32_t)(32 * wq) << 16);
        HbMomAcc acc;
        acc.clear();
        mbar_wait<false>(bar_w, 0);              // this CTA's weights are resident
        int stage = 0;
        uint32_t pin = 0, pd = 0;
        for (size_t g = cluster_id; g < ngroups; g += nclusters) {
            const size_t tile = g * CG + rank;
            const size_t i = tile * TILE_M + row;
            const bool valid = tile < ntiles && i < n;
            const bool full = tile < ntiles && (tile + 1) * TILE_M <= n;
            if (half == 0) {
                float c[6] = {0, 0, 0, 0, 0, 0};
                if (full) {
                    mbar_wait<false>(bar_in_full + 8 * stage, pin);
                    const float* st = reinterpret_cast<const float*>(smem + pl.stage_off + stage * STAGE_BYTES);
#pragma unroll
                    for (int j = 0; j < 6; ++j) c[j] = st[j * TILE_M + row];
                    __syncwarp();
                    if (lane == 0) mbar_arrive_local(bar_in_empty + 8 * stage);
                    stage ^= 1;
                    if (stage == 0) pin ^= 1;
                } else if (valid) {
#pragma unroll
                    for (int j = 0; j < 6; ++j) c[j] = p.v[j][i];
                }
                float nin[6] = {0, 0, 0, 0, 0, 0};
                if (valid) hb_sur_prologue(sd, c[0], c[1], c[2], c[3], c[4], c[5], nin);
                float lo[6];
#pragma unroll
                for (int j = 0; j < 6; ++j) lo[j] = nin[j] - round16<F16>(nin[j]);
                // K = 16 operand row: hi0..hi5, lo0..lo5, 0, 0, 0, 0  (two 16-byte chunks, swizzled)
                const uint32_t q0[4] = {pack2<F16>(nin[0], nin[1]), pack2<F16>(nin[2], nin[3]), pack2<F16>(nin[4], nin[5]),
                                        pack2<F16>(lo[0], lo[1])};
                const uint32_t q1[4] = {pack2<F16>(lo[2], lo[3]), pack2<F16>(lo[4], lo[5]), 0u, 0u};
                asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(a_row + ((0u ^ sw) << 4)), "r"(q0[0]), "r"(q0[1]), "r"(q0[2]), "r"(q0[3]) : "memory");
                asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(a_row + ((1u ^ sw) << 4)), "r"(q1[0]), "r"(q1[1]), "r"(q1[2]), "r"(q1[3]) : "memory");
            }
            fence_proxy_async();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive_cluster(bar_a, 0);

            for (int l = 0; l < pl.n_linear; ++l) {
                mbar_wait<false>(bar_d, pd);
                pd ^= 1;
                tc_fence_after();
                if (l < pl.n_linear - 1) {
                    const int npad = pl.npad[l];
                    const float* bl = bias_s + pl.bias_off[l];
                    const float slope = sd.prelu[l];
                    const int c_begin = half * (npad >> 1), c_end = c_begin + (npad >> 1);
                    for (int c0 = c_begin; c0 < c_end; c0 += 32) {
                        uint32_t r[32];
                        tmem_ld32(tlane + c0, r);
                        tmem_ld_wait();
                        uint32_t q[16];
#pragma unroll
                        for (int k = 0; k < 16; ++k) {
                            const float2 b2 = *reinterpret_cast<const float2*>(bl + c0 + 2 * k);
                            const float v0 = hb_activate<ACT, true>(__uint_as_float(r[2 * k]) + b2.x, slope);
                            const float v1 = hb_activate<ACT, true>(__uint_as_float(r[2 * k + 1]) + b2.y, slope);
                            q[k] = pack2<F16>(v0, v1);
                        }
                        const uint32_t slab = a_row + (c0 >> 6) * A_SLAB_BYTES;
                        const uint32_t ch0 = (uint32_t)((c0 & 63) >> 3);
#pragma unroll
                        for (int k = 0; k < 4; ++k)
                            asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(slab + (((ch0 + k) ^ sw) << 4)),
                                         "r"(q[4 * k]), "r"(q[4 * k + 1]), "r"(q[4 * k + 2]), "r"(q[4 * k + 3]) : "memory");
                    }
                    fence_proxy_async();
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) mbar_arrive_cluster(bar_a, 0);
                } else if (half == 0) {
                    uint32_t r[8];
                    tmem_ld8(tlane, r);
                    tmem_ld_wait();
                    tc_fence_before();
                    if (valid) {
                        const float* bl = bias_s + pl.bias_off[l];
                        float w[6];
#pragma unroll
                        for (int j = 0; j < 6; ++j) w[j] = __uint_as_float(r[j]) + bl[j];
                        float x, px, y, py, t, pt;
                        hb_sur_epilogue(sd, w, x, px, y, py, t, pt);
                        p.v[0][i] = x; p.v[1][i] = px; p.v[2][i] = y; p.v[3][i] = py; p.v[4][i] = t; p.v[5][i] = pt;
                        if (partials) acc.add(x, px, y, py, t, pt);
                    }
                }
            }
        }
        if (partials && half == 0) {
            double* red = reinterpret_cast<double*>(smem + pl.red_off);
            hb_block_reduce_moments(acc, red, partials + (size_t)blockIdx.x * HB_NMOM, tid - 64, 128, 2);
        }
    }
    // ---- teardown: everyone done with TMEM (both CTAs of a pair), then free it
    tc_fence_before();
    __syncthreads();
    if (CG == 2) cluster_sync_all();
    if (warp == 1) {
        tc_fence_after();
        tmem_dealloc<CG>(tmem_base, (uint32_t)pl.tmem_cols);
    }
}

// ------------------------------------------------------------------------------- host: plan + packing
int round_up(int v, int m) { return (v + m - 1) / m * m; }

void layer_geometry(int n_linear, const int* widths, int* kpad, int* npad, int* ksteps) {
    for (int l = 0; l < n_linear; ++l) {
        const bool last = l == n_linear - 1;
        npad[l] = last ? 16 : round_up(widths[l + 1], 64);
        if (l == 0) { kpad[l] = 64; ksteps[l] = 1; }                 // 6 hi + 6 lo + 4 zero
        else { kpad[l] = npad[l - 1]; ksteps[l] = npad[l - 1] / 16; }
    }
}

bool make_plan(int cg, int n_linear, const int* widths, TcPlan& pl) {
    std::memset(&pl, 0, sizeof pl);
    int kpad[HB_MAX_LINEAR], ksteps[HB_MAX_LINEAR];
    layer_geometry(n_linear, widths, kpad, pl.npad, ksteps);
    pl.n_linear = n_linear;
    int off = 0, boff = 0, maxslab = 1, maxn = 32;
    for (int l = 0; l < n_linear; ++l) {
        pl.ksteps[l] = ksteps[l];
        pl.nslab[l] = kpad[l] / 64;
        if ((pl.npad[l] / cg) % 8) return false;
        pl.w_slab_bytes[l] = pl.npad[l] / cg * 128;
        pl.w_off[l] = off;
        off += pl.nslab[l] * pl.w_slab_bytes[l];
        pl.bias_off[l] = boff;
        boff += pl.npad[l];
        if (pl.nslab[l] > maxslab) maxslab = pl.nslab[l];
        if (pl.npad[l] > maxn) maxn = pl.npad[l];
    }
    if (maxn > 512) return false;                                   // accumulator must fit the 512 TMEM columns
    if (cg == 2 && maxn > 256) return false;                        // pair mode: one N block (rows split 0..N/2 | N/2..N)
    pl.w_bytes_total = off;
    off = round_up(off, 1024);
    pl.a_off = off;
    off += maxslab * A_SLAB_BYTES;
    pl.stage_off = off;
    off += IN_STAGES * STAGE_BYTES;
    pl.bias_base = off;
    off += round_up(boff * 4, 16);
    pl.bar_off = off;
    off += 128;
    pl.red_off = off;
    off += 4 * HB_NMOM * 8;
    pl.total = off;
    int cols = 32;
    while (cols < maxn) cols <<= 1;
    pl.tmem_cols = cols;
    return (size_t)pl.total + 1024 <= SMEM_LIMIT;
}

template <int CG, int ACT, bool F16>
cudaError_t launch_one(const HbParticles& p, size_t n, const HbSurDev& sd, const TcPlan& pl, double* partials, int grid,
                       cudaStream_t s) {
    const size_t smem = (size_t)pl.total + 1024;   // slack so the 1024-byte alignment of the swizzle atoms always holds
    cudaError_t e = cudaFuncSetAttribute(hb_sur_tc_kernel<CG, ACT, F16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(THREADS);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = CG;
    at[0].val.clusterDim.y = 1;
    at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, hb_sur_tc_kernel<CG, ACT, F16>, p, n, sd, pl, partials);
}

template <int CG, bool F16>
cudaError_t launch_act(const HbParticles& p, size_t n, const HbSurDev& sd, const TcPlan& pl, double* partials, int grid,
                       cudaStream_t s) {
    switch (sd.act) {
    case 0: return launch_one<CG, 0, F16>(p, n, sd, pl, partials, grid, s);
    case 1: return launch_one<CG, 1, F16>(p, n, sd, pl, partials, grid, s);
    case 2: return launch_one<CG, 2, F16>(p, n, sd, pl, partials, grid, s);
    default: return launch_one<CG, 3, F16>(p, n, sd, pl, partials, grid, s);
    }
}

int choose_cg(int n_linear, const int* widths, TcPlan& pl) {
    // HB_TC_FORCE_CG=2 : test hook, runs shapes that fit one CTA on a CTA pair as well
    const char* force = getenv("HB_TC_FORCE_CG");
    if (force && force[0] == '2') return make_plan(2, n_linear, widths, pl) ? 2 : 0;
    if (make_plan(1, n_linear, widths, pl)) return 1;
    if (make_plan(2, n_linear, widths, pl)) return 2;
    return 0;
}

}  // namespace

bool hb_tc_supported(int prec, int n_linear, const int* widths, char* why, size_t why_len) {
    if (prec != 1 && prec != 2) {
        snprintf(why, why_len, "HB_PREC_TF32 has no kernel yet (use HB_PREC_BF16 or HB_PREC_F16)");
        return false;
    }
    TcPlan pl;
    if (!choose_cg(n_linear, widths, pl)) {
        snprintf(why, why_len, "weights do not fit resident in shared memory even split over a CTA pair "
                               "(or a hidden width exceeds 512); weight streaming is not built yet");
        return false;
    }
    return true;
}

// Packed operand image: per layer, per 64-wide K slab, npad rows of 128 bytes (K-major, 128-byte swizzle:
// the 16-byte chunk c of row r sits at chunk position c ^ (r mod 8)).  Layer 0 carries W_0 twice
// (columns 0..5 multiply the hi parts of the inputs, 6..11 the lo parts).
size_t hb_tc_pack_weights(int prec, int n_linear, const int* widths, const float* const* W, void* dst,
                          long long* off_bytes, int* kpad, int* npad) {
    int ksteps[HB_MAX_LINEAR];
    layer_geometry(n_linear, widths, kpad, npad, ksteps);
    size_t total = 0;
    for (int l = 0; l < n_linear; ++l) {
        off_bytes[l] = (long long)total;
        total += (size_t)(kpad[l] / 64) * npad[l] * 128;
    }
    if (!dst) return total;
    std::memset(dst, 0, total);
    unsigned char* base = static_cast<unsigned char*>(dst);
    for (int l = 0; l < n_linear; ++l) {
        const int fin = widths[l], fout = widths[l + 1];
        const int kcols = l == 0 ? 12 : fin;
        for (int o = 0; o < fout; ++o)
            for (int k = 0; k < kcols; ++k) {
                const float w = l == 0 ? W[l][(size_t)o * fin + (k % 6)] : W[l][(size_t)o * fin + k];
                const int slab = k / 64, kk = k % 64, c = kk / 8, e = kk % 8;
                const size_t byte = (size_t)off_bytes[l] + (size_t)slab * npad[l] * 128 + (size_t)o * 128 +
                                    (size_t)((c ^ (o & 7)) << 4) + (size_t)e * 2;
                unsigned short bits;
                if (prec == 2) { __half h = __float2half_rn(w); std::memcpy(&bits, &h, 2); }
                else { __nv_bfloat16 h = __float2bfloat16_rn(w); std::memcpy(&bits, &h, 2); }
                std::memcpy(base + byte, &bits, 2);
            }
    }
    return total;
}

cudaError_t hb_launch_sur_tc(const HbParticles& p, size_t n, const HbSurDev& sd, double* partials, int* nblocks_out,
                             int sm_count, cudaStream_t s) {
    TcPlan pl;
    const int cg = choose_cg(sd.n_linear, sd.widths, pl);
    if (cg == 0) return cudaErrorNotSupported;
    const size_t ntiles = (n + TILE_M - 1) / TILE_M;
    const size_t ngroups = (ntiles + cg - 1) / cg;
    size_t clusters = (size_t)(sm_count / cg);
    if (clusters > ngroups) clusters = ngroups;
    if (clusters < 1) clusters = 1;
    const int grid = (int)clusters * cg;
    if (nblocks_out) *nblocks_out = grid;
    const bool f16 = sd.prec == 2;
    if (cg == 1) return f16 ? launch_act<1, true>(p, n, sd, pl, partials, grid, s) : launch_act<1, false>(p, n, sd, pl, partials, grid, s);
    return f16 ? launch_act<2, true>(p, n, sd, pl, partials, grid, s) : launch_act<2, false>(p, n, sd, pl, partials, grid, s);
}
