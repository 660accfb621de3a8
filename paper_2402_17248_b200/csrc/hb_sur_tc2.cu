// hb_sur_tc2.cu -- surrogate stage on the 5th-gen tensor cores (HB_PREC_BF16 / HB_PREC_F16), weights resident in
// shared memory, every layer issued as two N-HALVES with their own accumulators: rows a4-a6 for nets whose hidden
// width is above 128 (C3: 6-256^3-6).
//
// Why.  hb_sur_tc.cu gives a 128-particle tile two full-width accumulator buffers (2 x 256 of the 512 TMEM columns)
// and packs the next layer's operand in place into the buffer it came from.  The tensor pipe then idles, once per
// layer, from "accumulator complete" until the epilogue warps have converted the first K slab (~600-900 cycles
// against 2100 cycles of MMAs), and at the tile boundary for the whole chain last hidden layer -> convert -> last
// layer -> output read (measured with a clock64 probe build, profiles/r2_mma_rate.md).  Here the 512 columns are cut differently:
//     A[0] = [0,128)   A[1] = [128,256)    packed 16-bit operands (256 values in 128 columns), ping-pong per layer
//     D[0] = [256,384) D[1] = [384,512)    fp32 accumulators of the two N-halves of the layer in flight
// and every layer goes out as two tcgen05.mma chains of N = width/2 (an N = 128 MMA runs at full rate: 67 cycles for
// M128 x N128 x K16 against 131 for N256, profiles/r2_mma_rate.md).  While half 1's MMAs run, the epilogue warps turn
// half 0's accumulator into K-half 0 of the next operand (written to the OTHER operand region: nothing is held in
// registers, nothing waits for the layer to end); the next layer's half 0 starts on that K-half the moment half 1's
// MMAs are through, and meets K-half 1 (converted from half 1 meanwhile) eight K steps later.  At the tile boundary the
// next tile's layer 0 (half 0) is issued right behind the last hidden layer, before the last layer (N = 16, into D[1]);
// only its half 1 waits for the output read.  (Measured and dropped: the 16 output columns in the dead operand region
// instead of D[1], so that no MMA waits for the output read: 2.40 ms against 2.20; and the next tile's first operand
// half converted under the last hidden layer with its K-half 0 issued before the last layer: 2.42 ms.  After the issuing
// warp's waits were changed -- hb_tc_common.cuh, mbar_spin: 2.20 -> 2.05 ms -- five more re-orderings of the tile boundary and
// of the epilogue were built, verified and measured slower: profiles/r2_issuer_codegen.md lists them with their times.)
// Events.  The hidden accumulators of a CTA form one sequence e = 0, 1, 2, ...: tile t, layer l <= L-2, half h is
// e = (t (L-1) + l) * 2 + h; it lives in D[h], signals DH_FULL[h], is read (DH_FREE[h]) and converted into K-half h of
// operand region (t (L-1) + l) & 1 (A_FULL[h]).
// Bias.  The layer-0 operand row is  hi0..5, lo0..5, 1, 1, 0, 0;  W_0 carries b_hi, b_lo in K columns 12, 13; every
// hidden half gets one extra K = 16 MMA (accumulate = 0) of that operand tile against its bias block.
// Warp roles (14 warps): 0-3 IO (a4 prologue of the next tile, a6 output + a3 moments of the current one), 4-11
// epilogue (lane quarter = warp % 4, column half = (warp - 4) / 4), 12 copy producer (weights once, then the six
// coordinate rows of every tile through the TMA engine), 13 MMA issuer (leader CTA of a pair, one elected lane).
#include "hb_tc_common.cuh"

namespace {

constexpr int T2_THREADS = 448;
constexpr int T2_STAGES = 2;          // input staging ring (tiles)
constexpr uint32_t T2_A = 0;          // operand regions A[0], A[1]: 128 columns each
constexpr uint32_t T2_D = 256;        // accumulators D[0], D[1]: 128 columns each

enum : int {
    T_W = 0,              // weights resident (local)
    T_IN_FULL = 1,        // [2] coordinate rows staged (local)
    T_IN_EMPTY = 3,       // [2] stage consumed by the 4 IO warps (local)
    T_A0_FULL = 5,        // [2] layer-0 operand written (leader; 4 IO warps x CG)
    T_DH_FULL = 7,        // [2] accumulator D[h] of a hidden event complete (both CTAs, MMA commit)
    T_DH_FREE = 9,        // [2] D[h] read by the epilogue warps (leader; 8 warps x CG)
    T_A_FULL = 11,        // [2] K-half h of the next operand written (leader; 8 warps x CG)
    T_D_LAST = 13,        // accumulator of the last layer complete (both CTAs, MMA commit)
    T_OUT_READ = 14,      // last layer's accumulator read by the IO warps (leader; 4 IO warps x CG)
    T_COUNT = 15
};

struct T2Plan {
    int n_linear;
    int npad[HB_MAX_LINEAR];          // padded fan-out of layer l (last layer: 16)
    int hw[HB_MAX_LINEAR];            // N of one MMA of layer l: npad / 2 (l <= L-2), npad (last layer)
    int w_off[HB_MAX_LINEAR];         // smem byte offset of layer l's weights (this CTA's rows)
    int w_slab_bytes[HB_MAX_LINEAR];  // this CTA's bytes of one K slab (l >= 1) or of the whole layer (l = 0)
    int nslab[HB_MAX_LINEAR];         // 64-wide K slabs of layer l (l >= 1)
    int wb_off[HB_MAX_LINEAR];        // 1 <= l <= L-2: bias block (K = 16 operand, this CTA's rows, halves in order)
    int wb_bytes[HB_MAX_LINEAR];
    int a0_off, stage_off, bias_base, bar_off, red_off, phc_off, total, w_bytes_total;
};

// 16 accumulator columns -> r[O .. O+16)   (array references and compile-time offsets only: the arrays stay in registers)
template <int O>
__device__ __forceinline__ void tmem_ld16o(uint32_t taddr, uint32_t (&r)[64]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
        : "=r"(r[O + 0]), "=r"(r[O + 1]), "=r"(r[O + 2]), "=r"(r[O + 3]), "=r"(r[O + 4]), "=r"(r[O + 5]), "=r"(r[O + 6]),
          "=r"(r[O + 7]), "=r"(r[O + 8]), "=r"(r[O + 9]), "=r"(r[O + 10]), "=r"(r[O + 11]), "=r"(r[O + 12]), "=r"(r[O + 13]),
          "=r"(r[O + 14]), "=r"(r[O + 15])
        : "r"(taddr) : "memory");
}
// 8 packed operand columns <- q[O .. O+8)
template <int O>
__device__ __forceinline__ void tmem_st8o(uint32_t taddr, const uint32_t (&q)[64]) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
                 ::"r"(taddr), "r"(q[O + 0]), "r"(q[O + 1]), "r"(q[O + 2]), "r"(q[O + 3]), "r"(q[O + 4]), "r"(q[O + 5]),
                   "r"(q[O + 6]), "r"(q[O + 7]) : "memory");
}
// chunk C (16 values of r) -> sigma -> 16 bit, packed IN PLACE into r[8 C .. 8 C + 8) (chunks in ascending order: every
// value is read before its register is reused)
template <int ACT, bool F16, int C>
__device__ __forceinline__ void t2_convert(uint32_t (&r)[64], float slope) {
#pragma unroll
    for (int k = 0; k < 8; ++k)
        r[8 * C + k] = act_pack<ACT, F16>(__uint_as_float(r[16 * C + 2 * k]), __uint_as_float(r[16 * C + 2 * k + 1]), slope);
}

// K = 16 steps [KB, KE) of one MMA chain, A from tensor memory (8 columns per step), B = K slab k / 4 of the half's weight
// rows, 32 bytes per step inside the slab.  Compile-time bounds, one straight-line run of MMAs: the issuing warp is a
// single thread of dependent instructions (~5 cycles each); with run-time bounds (predicated slots, or a loop with
// barrier probes in it) issuing costs ~60 cycles per MMA (measured, profiles/r2_mma_rate.md) -- as much as an N = 128 MMA
// takes to execute, and four times what the last layer's N = 16 MMAs take.
template <int CG, int KB, int KE>
__device__ __forceinline__ void t2_issue_range(uint32_t d_tmem, uint32_t a_tmem, uint64_t bd, uint64_t bd_step, uint32_t idesc,
                                               bool first_overwrites) {
#pragma unroll
    for (int k = KB; k < KE; ++k) {
        const uint64_t bs = bd + (uint64_t)(k >> 2) * bd_step + (uint64_t)(2 * (k & 3));
        if (k == 0) {
            if (first_overwrites) umma_ts<CG, false>(d_tmem, a_tmem, bs, idesc);
            else umma_ts<CG, true>(d_tmem, a_tmem, bs, idesc);
        } else {
            umma_ts<CG, true>(d_tmem, a_tmem + (uint32_t)(8 * k), bs, idesc);
        }
    }
}
// part 0: K-half 0 = steps [0, ksteps/2);  part 1: K-half 1;  part 2: all steps.  ksteps = 4, 8, 12 or 16 (widths pad to 64)
template <int CG>
__device__ __forceinline__ void t2_issue_ksteps(int part, int ksteps, uint32_t d_tmem, uint32_t a_tmem, uint64_t bd,
                                                uint64_t bd_step, uint32_t idesc, bool first_overwrites) {
#define T2_CASE(KS)                                                                                             \
    case KS:                                                                                                    \
        if (part == 0) t2_issue_range<CG, 0, KS / 2>(d_tmem, a_tmem, bd, bd_step, idesc, first_overwrites);      \
        else if (part == 1) t2_issue_range<CG, KS / 2, KS>(d_tmem, a_tmem, bd, bd_step, idesc, false);           \
        else t2_issue_range<CG, 0, KS>(d_tmem, a_tmem, bd, bd_step, idesc, first_overwrites);                    \
        break;
    switch (ksteps) {
        T2_CASE(4)
        T2_CASE(8)
        T2_CASE(12)
        default:
        T2_CASE(16)
    }
#undef T2_CASE
}

template <int CG, int ACT, bool F16>
__global__ void __launch_bounds__(T2_THREADS, 1)
hb_sur_tc2_kernel(HbParticles p, size_t n, const __grid_constant__ HbSurDev sd, const __grid_constant__ T2Plan pl,
                  double* __restrict__ partials) {
    constexpr int PROD_WARP = 12, MMA_WARP = 13;
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    // the 128-byte swizzle atoms (8 rows x 128 B) must sit on 1024-byte boundaries of the shared window
    unsigned char* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    const uint32_t sbase = smem_u32(smem);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const uint32_t rank = CG == 1 ? 0u : cluster_rank();
    const size_t ntiles = (n + TILE_M - 1) / TILE_M;
    const size_t ngroups = (ntiles + CG - 1) / CG;
    const size_t cluster_id = blockIdx.x / CG, nclusters = gridDim.x / CG;
    // tile groups of this CTA (pair): g_t = cluster_id + t * nclusters, t < nmine
    const uint32_t nmine = cluster_id < ngroups ? (uint32_t)((ngroups - cluster_id + nclusters - 1) / nclusters) : 0u;
    const int L = pl.n_linear;

    const uint32_t bar0 = sbase + pl.bar_off;
    auto bar = [&](int i) -> uint32_t { return bar0 + 8u * (uint32_t)i; };
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + pl.bar_off + 8 * T_COUNT);
    float* bias_s = reinterpret_cast<float*>(smem + pl.bias_base);

    if (tid == 0) {
        mbar_init(bar(T_W), 1);
        for (int s = 0; s < 2; ++s) {
            mbar_init(bar(T_IN_FULL + s), 1);
            mbar_init(bar(T_IN_EMPTY + s), 4);
            mbar_init(bar(T_A0_FULL + s), 4 * CG);
            mbar_init(bar(T_DH_FULL + s), 1);
            mbar_init(bar(T_DH_FREE + s), 8 * CG);
            mbar_init(bar(T_A_FULL + s), 8 * CG);
        }
        mbar_init(bar(T_D_LAST), 1);
        mbar_init(bar(T_OUT_READ), 4 * CG);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == MMA_WARP) {
        tmem_alloc<CG>(smem_u32(tmem_slot), 512u);
        tmem_relinquish<CG>();
    }
    // bias of the last layer -> shared (fp32, added by the IO warps); the other biases ride in the MMAs
    for (int i = tid; i < pl.npad[L - 1]; i += T2_THREADS) bias_s[i] = sd.btc[sd.btc_off[L - 1] + i];
    tc_fence_before();
    __syncthreads();
    if (CG == 2) cluster_sync_all();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    if (warp == PROD_WARP) {
        // ===================================================== producer: weights once, then particle tiles
        if (lane == 0) {
            mbar_expect_tx(bar(T_W), (uint32_t)pl.w_bytes_total);
            const unsigned char* wg = reinterpret_cast<const unsigned char*>(sd.wtc);
            bulk_g2s(sbase + pl.w_off[0], wg + sd.wtc_off[0] + (size_t)rank * pl.w_slab_bytes[0],
                     (uint32_t)pl.w_slab_bytes[0], bar(T_W));
            for (int l = 1; l < L; ++l) {
                const size_t slab_all = (size_t)pl.w_slab_bytes[l] * CG;           // one K slab, both ranks
                for (int s = 0; s < pl.nslab[l]; ++s)
                    bulk_g2s(sbase + pl.w_off[l] + s * pl.w_slab_bytes[l],
                             wg + sd.wtc_off[l] + (size_t)s * slab_all + (size_t)rank * pl.w_slab_bytes[l],
                             (uint32_t)pl.w_slab_bytes[l], bar(T_W));
                if (l + 1 < L)                                                      // bias block behind the K slabs
                    bulk_g2s(sbase + pl.wb_off[l],
                             wg + sd.wtc_off[l] + (size_t)pl.nslab[l] * slab_all + (size_t)rank * pl.wb_bytes[l],
                             (uint32_t)pl.wb_bytes[l], bar(T_W));
            }
            int stage = 0;
            uint32_t ph = 0;
            for (uint32_t t = 0; t < nmine; ++t) {
                const size_t tile = (cluster_id + (size_t)t * nclusters) * CG + rank;
                const bool full = tile < ntiles && (tile + 1) * TILE_M <= n;
                if (full) {
                    mbar_wait<false>(bar(T_IN_EMPTY + stage), ph ^ 1);
                    mbar_expect_tx(bar(T_IN_FULL + stage), STAGE_BYTES);
                    for (int j = 0; j < 6; ++j)
                        bulk_g2s(sbase + pl.stage_off + stage * STAGE_BYTES + j * TILE_M * 4, p.v[j] + tile * TILE_M,
                                 TILE_M * 4, bar(T_IN_FULL + stage));
                    stage ^= 1;
                    if (stage == 0) ph ^= 1;
                }
            }
        }
        __syncwarp();
    } else if (warp == MMA_WARP) {
        // ===================================================== MMA issuer (leader CTA of the pair only)
        // The whole warp walks the schedule (warp-uniform control flow, barrier waits by every lane); one elected
        // lane issues the MMAs and commits.
        if (rank == 0) {
            const uint32_t fmt = F16 ? 0u : 1u;
            const uint32_t idesc_base = (1u << 4) | (fmt << 7) | (fmt << 10) | ((uint32_t)((TILE_M * CG) >> 4) << 24);
            const bool issuer = elect_one();
            const uint32_t dbase = tmem_base + T2_D;     // D[h] = dbase + 128 h
            uint32_t ph_free = 0, ph_a = 0;        // bit h: parity of the next completion of DH_FREE[h] / A_FULL[h]
            uint32_t used = 0;                     // bit h: D[h] has held a hidden event before
            // Per-phase constants (phase = layer l >= 1, half h), built once into shared memory: between the last MMA of
            // one phase and the first MMA of the next the pipe only has the ~5 MMAs of its queue to run (~330 cycles at
            // N = 128), so whatever the issuer computes there (descriptors: dependent loads from the constant bank) is
            // tensor-pipe idle time.  entry 2 l + h: {B descriptor of the half, bias-block descriptor, idesc, K-slab step}
            uint4* phc = reinterpret_cast<uint4*>(smem + pl.phc_off);
            if (lane < 2 * L && lane >= 2) {
                const int l = lane >> 1, h = lane & 1;
                const uint32_t half_rows = (uint32_t)(h * (pl.hw[l] / CG));
                const uint64_t bd = make_desc(sbase + pl.w_off[l] + half_rows * 128u);
                const uint64_t wbd = make_desc_l0(sbase + pl.wb_off[l] + half_rows * 32u);
                phc[2 * lane] = make_uint4((uint32_t)bd, (uint32_t)(bd >> 32), (uint32_t)wbd, (uint32_t)(wbd >> 32));
                phc[2 * lane + 1] = make_uint4(idesc_base | ((uint32_t)(pl.hw[l] >> 3) << 17), (uint32_t)(pl.w_slab_bytes[l] >> 4),
                                               (uint32_t)(pl.npad[l - 1] >> 4), (uint32_t)(pl.npad[l - 1] >> 5));
            }
            __syncwarp();
            // D[h] is written again: the epilogue warps must have read the event it holds
            auto claim = [&](int h) {
                if ((used >> h) & 1u) {
                    mbar_spin(bar(T_DH_FREE + h), (ph_free >> h) & 1u);
                    ph_free ^= 1u << h;
                }
                used |= 1u << h;
            };
            const uint64_t w0d0 = make_desc_l0(sbase + pl.w_off[0]);
            const uint64_t w0d1 = make_desc_l0(sbase + pl.w_off[0] + (uint32_t)(pl.hw[0] / CG) * 32u);
            const uint32_t idesc0 = idesc_base | ((uint32_t)(pl.hw[0] >> 3) << 17);
            // layer 0 of tile t, half h: one K = 16 MMA from the compact operand (bias inside W_0)
            auto issue_l0 = [&](uint32_t t, int h) {
                if (h == 1) {
                    // D[1] holds the previous tile's outputs until the IO warps have read them (the last layer, not the
                    // epilogue, wrote it last: its DH_FREE phase was consumed by that layer)
                    if (t > 0) mbar_spin(bar(T_OUT_READ), (t - 1) & 1);
                    else used |= 2u;
                } else {
                    claim(0);
                    mbar_spin(bar(T_A0_FULL + (int)(t & 1)), (t >> 1) & 1);
                }
                tc_fence_after();
                if (issuer) {
                    umma<CG, false>(dbase + 128u * (uint32_t)h, make_desc_l0(sbase + pl.a0_off + (t & 1) * A0_BYTES),
                                    h ? w0d1 : w0d0, idesc0);
                    umma_commit<CG>(bar(T_DH_FULL + h));
                }
                __syncwarp();
            };
            if (nmine > 0) { issue_l0(0, 0); issue_l0(0, 1); }
            uint32_t lay = 0;                      // t (L-1) + l - 1: the operand region of layer l is lay & 1
            for (uint32_t t = 0; t < nmine; ++t) {
                const uint64_t a0d = make_desc_l0(sbase + pl.a0_off + (t & 1) * A0_BYTES);
                uint4 c0 = phc[4], c1 = phc[5];     // constants of the phase being issued (entry 2: layer 1, half 0)
                for (int l = 1; l < L; ++l, ++lay) {
                    const bool last = l == L - 1;
                    const uint32_t a_tmem = tmem_base + T2_A + 128u * (lay & 1u);
                    // before the last layer: the next tile's layer 0, half 0 (D[0] is free as soon as the epilogue has read
                    // the last hidden event in it; the operand region its epilogue writes is dead)
                    if (last && t + 1 < nmine) issue_l0(t + 1, 0);
                    for (int h = 0; h < (last ? 1 : 2); ++h) {
                        const uint32_t d_tmem = dbase + 128u * (uint32_t)(last ? 1 : h);   // the last layer's 16 columns go to D[1]
                        const uint64_t bd = ((uint64_t)c0.y << 32) | c0.x, wbd = ((uint64_t)c0.w << 32) | c0.z;
                        const uint32_t idesc = c1.x;
                        const uint64_t bd_step = c1.y;
                        const int ksteps = (int)c1.z;                    // K = 16 steps of the layer (K-half 1 starts at ksteps / 2)
                        // next phase's constants: in flight while this phase is issued
                        const int nxt = (h == 0 && !last) ? 2 * l + 1 : (l + 1 < L ? 2 * (l + 1) : 2);
                        c0 = phc[2 * nxt];
                        c1 = phc[2 * nxt + 1];
                        // What this phase waits for: its accumulator read by the epilogue (DH_FREE), and, for half 0 (and
                        // the last layer), the two K-halves of the operand the epilogue of layer l-1 is writing (A_FULL).
                        // Every wait on an mbarrier costs this warp ~165 cycles even when the phase completed long ago, so
                        // all three are probed at once first (lane i tests barrier i; test_wait does not suspend) and only
                        // what is really missing is awaited.
                        const int dh = last ? 1 : h;
                        const bool need_free = ((used >> dh) & 1u) != 0u, fresh = h == 0;
                        used |= 1u << dh;
                        uint32_t pbar = bar(T_DH_FREE + dh), ppar = (ph_free >> dh) & 1u;
                        if (lane == 1) { pbar = bar(T_A_FULL); ppar = ph_a & 1u; }
                        if (lane == 2) { pbar = bar(T_A_FULL + 1); ppar = (ph_a >> 1) & 1u; }
                        const bool probe = lane == 0 ? need_free : (lane < 3 && fresh);
                        const uint32_t have = __ballot_sync(0xffffffffu, probe && mbar_test(pbar, ppar) != 0u);
                        if (need_free) {
                            if (!(have & 1u)) mbar_spin(bar(T_DH_FREE + dh), (ph_free >> dh) & 1u);
                            ph_free ^= 1u << dh;
                        }
                        tc_fence_after();
                        // hidden layer: the bias goes in first, as one K = 16 MMA of the tile's layer-0 operand (ones in
                        // columns 12, 13) with this half's bias block (b_hi, b_lo in columns 12, 13, zeros elsewhere)
                        if (!last && issuer) umma<CG, false>(d_tmem, a0d, wbd, idesc);
                        if (fresh) {
                            // the operand is being written by the epilogue of layer l-1: K-half by K-half
                            if ((have & 6u) == 6u) {
                                if (issuer) t2_issue_ksteps<CG>(2, ksteps, d_tmem, a_tmem, bd, bd_step, idesc, last);
                            } else {
                                if (!(have & 2u)) {
                                    mbar_spin(bar(T_A_FULL), ph_a & 1u);
                                    tc_fence_after();
                                }
                                if (issuer) t2_issue_ksteps<CG>(0, ksteps, d_tmem, a_tmem, bd, bd_step, idesc, last);
                                mbar_spin(bar(T_A_FULL + 1), (ph_a >> 1) & 1u);
                                tc_fence_after();
                                if (issuer) t2_issue_ksteps<CG>(1, ksteps, d_tmem, a_tmem, bd, bd_step, idesc, false);
                            }
                            ph_a ^= 3u;
                        } else if (issuer) {
                            t2_issue_ksteps<CG>(2, ksteps, d_tmem, a_tmem, bd, bd_step, idesc, false);
                        }
                        if (issuer) umma_commit<CG>(bar(last ? T_D_LAST : T_DH_FULL + h));
                        __syncwarp();
                    }
                }
                if (t + 1 < nmine) issue_l0(t + 1, 1);
            }
        }
        __syncwarp();
    } else if (warp < EPI_WARP0) {
        // ===================================================== IO warps: prologue of tile t+1, output of tile t
        const int wq = warp & 3;                 // TMEM lane quarter this warp may access
        const int row = 32 * wq + lane;          // tile row = TMEM lane = particle within the tile
        const uint32_t a0_row = sbase + pl.a0_off + (uint32_t)(row >> 3) * 256 + (uint32_t)(row & 7) * 16;
        const uint32_t tout = tmem_base + ((uint32_t)(32 * wq) << 16) + T2_D + 128u;     // D[1], columns 0..7
        const float* bl = bias_s;
        HbMomAcc acc;
        acc.clear();
        int stage = 0;
        uint32_t pin = 0;
        // a4: load, convert, normalise, split, write the layer-0 operand of tile t
        auto prologue = [&](uint32_t t) {
            const size_t tile = (cluster_id + (size_t)t * nclusters) * CG + rank;
            const size_t i = tile * TILE_M + row;
            const bool valid = tile < ntiles && i < n;
            const bool full = tile < ntiles && (tile + 1) * TILE_M <= n;
            float c[6] = {0, 0, 0, 0, 0, 0};
            if (full) {
                mbar_wait<false>(bar(T_IN_FULL + stage), pin);
                const float* st = reinterpret_cast<const float*>(smem + pl.stage_off + stage * STAGE_BYTES);
#pragma unroll
                for (int j = 0; j < 6; ++j) c[j] = st[j * TILE_M + row];
                __syncwarp();
                if (lane == 0) mbar_arrive_local(bar(T_IN_EMPTY + stage));
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
            // K = 16 operand row: hi0..hi5, lo0..lo5, 1, 1, 0, 0  (two 16-byte chunks, 128 B apart); the ones meet
            // b_hi, b_lo in columns 12, 13 of the weights (layer 0) and of the bias blocks (hidden layers)
            const uint32_t q0[4] = {pack2<F16>(nin[0], nin[1]), pack2<F16>(nin[2], nin[3]), pack2<F16>(nin[4], nin[5]),
                                    pack2<F16>(lo[0], lo[1])};
            const uint32_t q1[4] = {pack2<F16>(lo[2], lo[3]), pack2<F16>(lo[4], lo[5]), pack2<F16>(1.0f, 1.0f), 0u};
            const uint32_t dst = a0_row + (t & 1u) * A0_BYTES;
            sts128(dst, q0);
            sts128(dst + 128, q1);
            fence_proxy_async();
            __syncwarp();
            if (lane == 0) mbar_arrive_cluster(bar(T_A0_FULL + (int)(t & 1u)), 0);
        };
        mbar_wait<false>(bar(T_W), 0);           // this CTA's weights are resident before the first MMA may start
        if (nmine > 0) prologue(0);
        for (uint32_t t = 0; t < nmine; ++t) {
            // operand buffer (t + 1) & 1 was last read by the bias MMAs of tile t - 1, complete before its output was
            if (t + 1 < nmine) prologue(t + 1);
            const size_t tile = (cluster_id + (size_t)t * nclusters) * CG + rank;
            const size_t i = tile * TILE_M + row;
            const bool valid = tile < ntiles && i < n;
            mbar_wait<true>(bar(T_D_LAST), t & 1);    // on the tile-boundary chain: the plain try_wait wakes sooner (2.063 -> 2.052 ms)
            tc_fence_after();
            uint32_t r[8];
            // the last layer read operand region (t (L-1) + L-2) & 1 and wrote the tail of the other one
            tmem_ld8(tout, r);
            tmem_ld_wait();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive_cluster(bar(T_OUT_READ), 0);
            if (valid) {
                float w[6];
#pragma unroll
                for (int j = 0; j < 6; ++j) w[j] = __uint_as_float(r[j]) + bl[j];
                float x, px, y, py, tt, pt;
                hb_sur_epilogue(sd, w, x, px, y, py, tt, pt);
                p.v[0][i] = x; p.v[1][i] = px; p.v[2][i] = y; p.v[3][i] = py; p.v[4][i] = tt; p.v[5][i] = pt;
                if (partials) acc.add(sd.mom_pivot, x, px, y, py, tt, pt);
            }
        }
        if (partials) {
            double* red = reinterpret_cast<double*>(smem + pl.red_off);
            hb_block_reduce_moments(acc, red, partials + blockIdx.x, tid - 32 * IO_WARP0, 128, 2);
        }
    } else {
        // ===================================================== epilogue warps: hidden events in issue order
        const int wq = warp & 3;
        const int grp = (warp - EPI_WARP0) >> 2;  // which half of an event's accumulator columns this warp converts
        const uint32_t tlane = tmem_base + ((uint32_t)(32 * wq) << 16);
        const uint32_t nev = nmine * (uint32_t)(L - 1) * 2u;
        uint32_t ph_full = 0;                     // bit h: parity of the next completion of DH_FULL[h]
        uint32_t lay = 0;                         // t (L-1) + l of the event
        int l = 0;
        auto arrive = [&](int b) {
            __syncwarp();
            if (lane == 0) mbar_arrive_cluster(bar(b), 0);
        };
        for (uint32_t e = 0; e < nev; ++e) {
            const int h = (int)(e & 1u);
            const float slope = sd.prelu[l];
            const int hwl = pl.npad[l] >> 1;      // accumulator columns of one half of layer l
            const int cw = hwl >> 1;              // ... of which this warp converts cw, as nch chunks of 16
            const int nch = cw >> 4;
            const uint32_t src = tlane + T2_D + 128u * (uint32_t)h + (uint32_t)(grp * cw);
            // K-half h of the next operand, in the region the layer before did NOT read
            const uint32_t dst = tlane + T2_A + 128u * (lay & 1u) + (uint32_t)(h * (hwl >> 1) + grp * (cw >> 1));
            mbar_wait<true>(bar(T_DH_FULL + h), (ph_full >> h) & 1u);
            ph_full ^= 1u << h;
            tc_fence_after();
            uint32_t r[64];
            if (nch > 0) tmem_ld16o<0>(src, r);
            if (nch > 1) tmem_ld16o<16>(src + 16u, r);
            if (nch > 2) tmem_ld16o<32>(src + 32u, r);
            if (nch > 3) tmem_ld16o<48>(src + 48u, r);
            tmem_ld_wait();
            tc_fence_before();
            arrive(T_DH_FREE + h);                // the accumulator may be overwritten
            if (nch > 0) t2_convert<ACT, F16, 0>(r, slope);
            if (nch > 1) t2_convert<ACT, F16, 1>(r, slope);
            if (nch > 2) t2_convert<ACT, F16, 2>(r, slope);
            if (nch > 3) t2_convert<ACT, F16, 3>(r, slope);
            if (nch > 0) tmem_st8o<0>(dst, r);
            if (nch > 1) tmem_st8o<8>(dst + 8u, r);
            if (nch > 2) tmem_st8o<16>(dst + 16u, r);
            if (nch > 3) tmem_st8o<24>(dst + 24u, r);
            tmem_st_wait();
            tc_fence_before();
            arrive(T_A_FULL + h);
            if (h == 1) {
                ++lay;
                if (++l == L - 1) l = 0;
            }
        }
    }
    // ---- teardown: everyone done with TMEM (both CTAs of a pair), then free it
    tc_fence_before();
    __syncthreads();
    if (CG == 2) cluster_sync_all();
    if (warp == MMA_WARP) {
        tc_fence_after();
        tmem_dealloc<CG>(tmem_base, 512u);
    }
}

// ------------------------------------------------------------------------------- host: plan, packing, launch
int t2_round_up(int v, int m) { return (v + m - 1) / m * m; }

bool t2_make_plan(int cg, int n_linear, const int* widths, T2Plan& pl) {
    std::memset(&pl, 0, sizeof pl);
    if (n_linear < 2 || n_linear > HB_MAX_LINEAR) return false;
    pl.n_linear = n_linear;
    int off = 0;
    for (int l = 0; l < n_linear; ++l) {
        const bool last = l == n_linear - 1;
        pl.npad[l] = last ? 16 : t2_round_up(widths[l + 1], 64);
        if (pl.npad[l] > 256) return false;                          // operand <= 128 columns, half accumulator <= 128
        pl.hw[l] = last ? pl.npad[l] : pl.npad[l] / 2;
        if ((pl.hw[l] / cg) % 8) return false;
        pl.nslab[l] = l == 0 ? 0 : pl.npad[l - 1] / 64;
        pl.w_slab_bytes[l] = pl.npad[l] / cg * (l == 0 ? 32 : 128);
        pl.w_off[l] = off;
        off += (l == 0 ? 1 : pl.nslab[l]) * pl.w_slab_bytes[l];
        pl.w_bytes_total += (l == 0 ? 1 : pl.nslab[l]) * pl.w_slab_bytes[l];
        if (l >= 1 && !last) {
            pl.wb_off[l] = off;
            pl.wb_bytes[l] = pl.npad[l] / cg * 32;
            off += pl.wb_bytes[l];
            pl.w_bytes_total += pl.wb_bytes[l];
        }
        off = t2_round_up(off, 1024);
    }
    pl.a0_off = off;
    off += 2 * A0_BYTES;
    pl.stage_off = off;
    off += T2_STAGES * STAGE_BYTES;
    pl.bias_base = off;
    off += t2_round_up(pl.npad[n_linear - 1] * 4, 16);
    pl.bar_off = off;
    off += t2_round_up(8 * T_COUNT + 8, 16);
    pl.red_off = off;
    off += 4 * HB_NMOM * 8;
    pl.phc_off = off;
    off += 2 * HB_MAX_LINEAR * 32;
    pl.total = off;
    return (size_t)pl.total + 1024 <= SMEM_LIMIT;
}

template <int CG, int ACT, bool F16>
cudaError_t t2_launch_one(const HbParticles& p, size_t n, const HbSurDev& sd, const T2Plan& pl, double* partials, int grid,
                          bool prepare, cudaStream_t s) {
    const size_t smem = (size_t)pl.total + 1024;   // slack so the 1024-byte alignment of the swizzle atoms always holds
    if (prepare)
        return cudaFuncSetAttribute(hb_sur_tc2_kernel<CG, ACT, F16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(T2_THREADS);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = CG;
    at[0].val.clusterDim.y = 1;
    at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, hb_sur_tc2_kernel<CG, ACT, F16>, p, n, sd, pl, partials);
}

template <int CG, bool F16>
cudaError_t t2_launch_act(const HbParticles& p, size_t n, const HbSurDev& sd, const T2Plan& pl, double* partials, int grid,
                          bool prepare, cudaStream_t s) {
    switch (sd.act) {
    case 0: return t2_launch_one<CG, 0, F16>(p, n, sd, pl, partials, grid, prepare, s);
    case 1: return t2_launch_one<CG, 1, F16>(p, n, sd, pl, partials, grid, prepare, s);
    case 2: return t2_launch_one<CG, 2, F16>(p, n, sd, pl, partials, grid, prepare, s);
    default: return t2_launch_one<CG, 3, F16>(p, n, sd, pl, partials, grid, prepare, s);
    }
}

}  // namespace

// 0: no plan; else the cluster size (1: the whole net fits one CTA, 2: CTA pair, each CTA holds half of every B operand)
int hb_tc2_plan_cg(int n_linear, const int* widths, int force_cg) {
    T2Plan pl;
    int maxn = 0;
    for (int l = 1; l < n_linear; ++l) maxn = widths[l] > maxn ? widths[l] : maxn;
    if (maxn <= 128) return 0;                   // narrow nets: two CTAs per SM on hb_sur_tc.cu do the same job
    if (force_cg != 2 && t2_make_plan(1, n_linear, widths, pl)) return 1;
    if (t2_make_plan(2, n_linear, widths, pl)) return 2;
    return 0;
}

// Packed operand image of this kernel.  Per layer [rank 0 | rank 1] blocks (one block for cg = 1):
//   Row order of every layer but the last: local row h (hw/cg) + i of rank r is neuron h hw + r (hw/cg) + i, hw = npad/2:
//     the rows of N-half 0 first, then those of N-half 1 (a cta_group::2 MMA of N = hw takes hw/2 rows from each CTA).
//   layer 0 (K = 16, no swizzle): per 8-row group 256 bytes = K chunk 0 of the 8 rows (8 x 16 B), then K chunk 1; W_0 is
//     carried twice (columns 0..5 meet the hi parts of the inputs, 6..11 the lo parts), b_hi, b_lo in columns 12, 13.
//   hidden layer l: per 64-wide K slab, per rank npad/cg rows of 128 bytes (K-major, 128-byte swizzle: the 16-byte chunk
//     c of local row i sits at chunk position c ^ (i mod 8)).  Behind the slabs the bias block (K = 16 operand as
//     layer 0, same row order).
//   last layer: per K slab, per rank 16/cg rows.
size_t hb_tc2_pack_weights(int prec, int cg, int n_linear, const int* widths, const float* const* W, const float* const* B,
                           void* dst, long long* off_bytes, int* kpad, int* npad) {
    T2Plan pl;
    if (!t2_make_plan(cg, n_linear, widths, pl)) return 0;
    size_t total = 0;
    for (int l = 0; l < n_linear; ++l) {
        off_bytes[l] = (long long)total;
        npad[l] = pl.npad[l];
        kpad[l] = l == 0 ? 16 : pl.npad[l - 1];
        total += (size_t)cg * ((size_t)(l == 0 ? 1 : pl.nslab[l]) * pl.w_slab_bytes[l] + pl.wb_bytes[l]);
        total = (total + 15) / 16 * 16;
    }
    if (!dst) return total;
    std::memset(dst, 0, total);
    unsigned char* base = static_cast<unsigned char*>(dst);
    auto bits16 = [prec](float w) {
        unsigned short bits;
        if (prec == 2) { __half h = __float2half_rn(w); std::memcpy(&bits, &h, 2); }
        else { __nv_bfloat16 h = __float2bfloat16_rn(w); std::memcpy(&bits, &h, 2); }
        return bits;
    };
    auto back32 = [prec](unsigned short bits) {
        if (prec == 2) { __half h; std::memcpy(&h, &bits, 2); return __half2float(h); }
        __nv_bfloat16 h; std::memcpy(&h, &bits, 2); return __bfloat162float(h);
    };
    auto put = [&](size_t byte, float w) { const unsigned short b = bits16(w); std::memcpy(base + byte, &b, 2); };
    for (int l = 0; l < n_linear; ++l) {
        const bool last = l == n_linear - 1;
        const int fin = widths[l], fout = widths[l + 1];
        const int rows = pl.npad[l] / cg, hr = pl.hw[l] / cg;       // rows per rank; rows per rank and N-half
        for (int o = 0; o < fout; ++o) {
            // neuron o -> (rank, local row)
            const int h = o / pl.hw[l], within = o % pl.hw[l];
            const int rank = within / hr, i = h * hr + within % hr;
            if (l == 0) {
                const size_t blk = (size_t)off_bytes[0] + (size_t)rank * pl.w_slab_bytes[0];
                const size_t rowb = blk + (size_t)(i / 8) * 256 + (size_t)(i % 8) * 16;
                for (int k = 0; k < 12; ++k) put(rowb + (size_t)(k / 8) * 128 + (size_t)(k % 8) * 2, W[0][(size_t)o * fin + (k % 6)]);
                const unsigned short hi = bits16(B[0][o]);
                put(rowb + 128 + 4 * 2, B[0][o]);                                   // k = 12
                put(rowb + 128 + 5 * 2, B[0][o] - back32(hi));                      // k = 13
            } else {
                const size_t slab_all = (size_t)pl.w_slab_bytes[l] * cg;
                for (int k = 0; k < fin; ++k) {
                    const int s = k / 64, kk = k % 64, c = kk / 8, e = kk % 8;
                    put((size_t)off_bytes[l] + (size_t)s * slab_all + (size_t)rank * pl.w_slab_bytes[l] + (size_t)i * 128 +
                            (size_t)((c ^ (i & 7)) << 4) + (size_t)e * 2,
                        W[l][(size_t)o * fin + k]);
                }
                if (!last) {
                    const size_t blk = (size_t)off_bytes[l] + (size_t)pl.nslab[l] * slab_all + (size_t)rank * pl.wb_bytes[l];
                    const size_t rowb = blk + (size_t)(i / 8) * 256 + (size_t)(i % 8) * 16;
                    const unsigned short hi = bits16(B[l][o]);
                    put(rowb + 128 + 4 * 2, B[l][o]);
                    put(rowb + 128 + 5 * 2, B[l][o] - back32(hi));
                }
            }
        }
        (void)rows;
    }
    return total;
}

// prepare: only set the kernel's shared-memory attribute (hb_lattice_finalize), launch nothing
cudaError_t hb_launch_sur_tc2(const HbParticles& p, size_t n, const HbSurDev& sd, double* partials, int* nblocks_out,
                              int sm_count, bool prepare, cudaStream_t s) {
    T2Plan pl;
    const int cg = sd.tc_cg;
    if ((cg != 1 && cg != 2) || !t2_make_plan(cg, sd.n_linear, sd.widths, pl)) return cudaErrorNotSupported;
    const size_t ntiles = (n + TILE_M - 1) / TILE_M;
    const size_t ngroups = (ntiles + cg - 1) / cg;
    size_t clusters = (size_t)(sm_count / cg);
    if (clusters > ngroups) clusters = ngroups;
    if (clusters < 1) clusters = 1;
    const int grid = (int)clusters * cg;
    if (nblocks_out) *nblocks_out = grid;
    const bool f16 = sd.prec == 2;
    if (cg == 1) return f16 ? t2_launch_act<1, true>(p, n, sd, pl, partials, grid, prepare, s)
                            : t2_launch_act<1, false>(p, n, sd, pl, partials, grid, prepare, s);
    return f16 ? t2_launch_act<2, true>(p, n, sd, pl, partials, grid, prepare, s)
               : t2_launch_act<2, false>(p, n, sd, pl, partials, grid, prepare, s);
}
