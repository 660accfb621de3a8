// hb_sur_tc2.cu -- surrogate stage on the 5th-gen tensor cores (HB_PREC_BF16 / HB_PREC_F16), weights resident in
// shared memory, TWO 128-particle tiles in flight per CTA (256 per CTA pair): rows a4-a6 for nets whose hidden
// width is above 128 (C3: 6-256^3-6).
//
// Why.  hb_sur_tc.cu keeps one tile per CTA in tensor memory: a 128 x 256 fp32 accumulator is 256 of the 512 TMEM
// columns and the next layer's operand is packed in place into the accumulator it came from, so the second
// accumulator buffer belongs to the same tile and the tensor pipe idles, once per layer, for the whole hand-over
// (commit -> epilogue wake -> convert -> arrive -> issue: ~900 cycles against 2048 cycles of MMAs, profiles/).
// Here a tile owns 256 columns: its packed 16-bit operand in columns [0,128) and HALF an accumulator in [128,256).
// Every hidden layer is issued as two N-halves (tcgen05.mma with N = width/2: measured at full rate, 67 cycles for
// M128 x N128 x K16 against 131 for N256, profiles/r2_mma_rate.md), both halves into the same 128 columns:
//     half 0 complete -> the epilogue warps read it, convert it and HOLD the packed result in registers (the operand
//                        columns are still being read by half 1's MMAs) -> half 1 may overwrite the accumulator;
//     half 1 complete -> the layer's operand is dead: the held half goes to operand columns [0,64), half 1 is read,
//                        converted and stored to [64,128): the next layer's operand, K-half by K-half.
// Two such tiles (slots) are in flight, each a pipeline of its own: its own MMA-issuing warp, its own four epilogue
// warps, its own barriers.  tcgen05.mma is accepted by the tensor pipe one at a time (measured: an issuing thread runs
// in lock step with the pipe, there is no deep queue), so whatever the issuer of a slot does between two phases --
// barrier waits, descriptors, ~800 cycles -- would leave the pipe idle; with two issuing warps the pipe takes the other
// slot's MMAs meanwhile.  Nothing orders the two slots against each other but the IO warps, which serve tiles in turn.
// Phases of a tile (L linear maps, L >= 2):
//     a          layer 0, one MMA (K = 16, N = npad_0) from the compact shared-memory operand into columns [0,npad_0)
//                of the slot (operand + accumulator columns: the slot holds no operand yet); bias inside (W_0 carries
//                b_hi, b_lo in K columns 12, 13; the operand row carries ones there)
//     (l,0),(l,1) hidden layer l = 1..L-2, N-half h: one K = 16 bias MMA (accumulate = 0: the tile's layer-0 operand
//                against the half's bias block) + npad_{l-1}/16 MMAs with A from tensor memory
//     d          last layer (N = 16), A from tensor memory; its bias is added in fp32 by the IO warps
// Warp roles (15 warps): 0-3 IO (a4 prologue of the tile after next, a6 output + a3 moments of the current one),
// 4-7 / 8-11 hidden-layer epilogue of slot 0 / 1 (lane quarter = warp % 4), 12 copy producer (weights once, then the six
// coordinate rows of every tile through the TMA engine into a 4-stage ring), 13 / 14 MMA issuer of slot 0 / 1 (leader CTA).
#include "hb_tc_common.cuh"

namespace {

constexpr int T2_THREADS = 480;
constexpr int T2_STAGES = 4;          // input staging ring (tiles)
constexpr uint32_t T2_SLOT_COLS = 256;  // TMEM columns of one tile slot
constexpr uint32_t T2_DH = 128;       // first accumulator column of a slot (the operand lives below it)

enum : int {
    T_W = 0,              // weights resident (local)
    T_IN_FULL = 1,        // [T2_STAGES] coordinate rows staged (local)
    T_IN_EMPTY = 5,       // [T2_STAGES] stage consumed by the 4 IO warps (local)
    T_SLOT = 9,           // per slot: 8 barriers
    T_COUNT = 25
};
enum : int {              // offsets inside a slot's barrier block
    S_A0_FULL = 0,        // [2] layer-0 operand written (leader; 4 IO warps x CG)
    S_DH_FULL = 2,        // accumulator of phase a / (l,h) complete (both CTAs, MMA commit)
    S_DH_FREE = 3,        // accumulator read by the slot's epilogue warps (leader; 4 warps x CG)
    S_A_FULL = 4,         // [2] K-half of the next operand written (leader; 4 warps x CG)
    S_D_LAST = 6,         // accumulator of phase d complete (both CTAs, MMA commit)
    S_OUT_READ = 7        // phase d's accumulator read by the IO warps (leader; 4 IO warps x CG)
};

struct T2Plan {
    int n_linear;
    int npad[HB_MAX_LINEAR];          // padded fan-out of layer l (last layer: 16)
    int hw[HB_MAX_LINEAR];            // N of one MMA of layer l: npad (l = 0, l = L-1), npad / 2 (hidden)
    int w_off[HB_MAX_LINEAR];         // smem byte offset of layer l's weights (this CTA's rows)
    int w_slab_bytes[HB_MAX_LINEAR];  // this CTA's bytes of one K slab (l >= 1) or of the whole layer (l = 0)
    int nslab[HB_MAX_LINEAR];         // 64-wide K slabs of layer l (l >= 1)
    int wb_off[HB_MAX_LINEAR];        // 1 <= l <= L-2: bias block (K = 16 operand, this CTA's rows, halves in order)
    int wb_bytes[HB_MAX_LINEAR];
    int a0_off, stage_off, bias_base, bar_off, red_off, total, w_bytes_total;
};

// 16 accumulator columns -> r[O .. O+16)   (array references and compile-time offsets only: the arrays stay in registers)
template <int O>
__device__ __forceinline__ void tmem_ld16o(uint32_t taddr, uint32_t (&r)[16]) {
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
// 16 accumulator columns -> sigma -> 16 bit, packed into q[O .. O+8)
template <int ACT, bool F16, int O>
__device__ __forceinline__ void t2_convert(const uint32_t (&r)[16], float slope, uint32_t (&q)[64]) {
#pragma unroll
    for (int k = 0; k < 8; ++k)
        q[O + k] = act_pack<ACT, F16>(__uint_as_float(r[2 * k]), __uint_as_float(r[2 * k + 1]), slope);
}
// nch chunks (<= 8) of 8 packed operand columns <- registers (no wait)
__device__ __forceinline__ void t2_store(uint32_t taddr, int nch, const uint32_t (&q)[64]) {
    if (nch > 0) tmem_st8o<0>(taddr, q);
    if (nch > 1) tmem_st8o<8>(taddr + 8u, q);
    if (nch > 2) tmem_st8o<16>(taddr + 16u, q);
    if (nch > 3) tmem_st8o<24>(taddr + 24u, q);
    if (nch > 4) tmem_st8o<32>(taddr + 32u, q);
    if (nch > 5) tmem_st8o<40>(taddr + 40u, q);
    if (nch > 6) tmem_st8o<48>(taddr + 48u, q);
    if (nch > 7) tmem_st8o<56>(taddr + 56u, q);
}

// One phase (a or (l,h)) of its slot, seen by one epilogue warp (lane quarter wq of the tile): `sbar0` = address of the
// slot's barrier block, `tl` = TMEM address of the slot's column 0 in this warp's lanes, `hold` = the held half.
template <int ACT, bool F16>
__device__ __forceinline__ void t2_epilogue_phase(const HbSurDev& sd, const T2Plan& pl, uint32_t sbar0, uint32_t tl, int ph,
                                                  uint32_t parity, int lane, uint32_t (&hold)[64]) {
    auto sbar = [&](int i) -> uint32_t { return sbar0 + 8u * (uint32_t)i; };
    auto arrive = [&](int i) {
        __syncwarp();
        if (lane == 0) mbar_arrive_cluster(sbar(i), 0);
    };
    const int l = ph == 0 ? 0 : 1 + ((ph - 1) >> 1);
    const int h = ph == 0 ? 0 : ((ph - 1) & 1);
    const float slope = sd.prelu[l];
    const int hwl = pl.npad[l] >> 1;      // accumulator columns of one half of layer l: nch chunks of 16
    const int nch = hwl >> 4;
    const uint32_t acc0 = ph == 0 ? tl : tl + T2_DH;          // phase a: the accumulator starts at column 0
    mbar_wait<true>(sbar(S_DH_FULL), parity);
    tc_fence_after();
    uint32_t ra[16], rb[16];
    const uint32_t a_lo = tl;                                 // operand columns of K-half 0
    const uint32_t a_hi = tl + (uint32_t)(hwl >> 1);          // ... of K-half 1
    // hwl accumulator columns starting at SRC -> sigma -> 16 bit, packed into DST[0 .. hwl/2): chunks of 16 columns, the
    // next chunk's tcgen05.ld in flight while one is converted (two chunks + the 64 held registers: 128 registers per
    // thread is all a 15-warp CTA gets); every column has been read when it is through (tcgen05.wait::ld)
#define T2_PAIR(SRC, DST, C)                                                   \
    if (nch > (C)) {                                                           \
        tmem_ld_wait();                                                        \
        if (nch > (C) + 1) tmem_ld16o<0>((SRC) + 16u * ((C) + 1), rb);         \
        t2_convert<ACT, F16, 8 * (C)>(ra, slope, (DST));                       \
    }                                                                          \
    if (nch > (C) + 1) {                                                       \
        tmem_ld_wait();                                                        \
        if (nch > (C) + 2) tmem_ld16o<0>((SRC) + 16u * ((C) + 2), ra);         \
        t2_convert<ACT, F16, 8 * (C) + 8>(rb, slope, (DST));                   \
    }
#define T2_READ_CONVERT(SRC, DST)                              \
    do {                                                       \
        tmem_ld16o<0>((SRC), ra);                              \
        T2_PAIR(SRC, DST, 0)                                   \
        T2_PAIR(SRC, DST, 2)                                   \
        T2_PAIR(SRC, DST, 4)                                   \
        T2_PAIR(SRC, DST, 6)                                   \
    } while (0)
    // `hold` doubles as the staging array of every conversion (it is dead outside the span half 0 -> half 1 of a hidden
    // layer)
    if (ph == 0) {
        // half 0 of layer 0's accumulator sits in the operand columns themselves; this warp alone touches its lanes, and
        // it has read all of half 0 before it writes
        T2_READ_CONVERT(acc0, hold);
        tc_fence_before();
        t2_store(a_lo, nch, hold);
        tmem_st_wait();
        tc_fence_before();
        arrive(S_A_FULL);
        T2_READ_CONVERT(acc0 + (uint32_t)hwl, hold);
        tc_fence_before();
        arrive(S_DH_FREE);
        t2_store(a_hi, nch, hold);
        tmem_st_wait();
        tc_fence_before();
        arrive(S_A_FULL + 1);
    } else if (h == 0) {
        T2_READ_CONVERT(acc0, hold);
        tc_fence_before();
        arrive(S_DH_FREE);                // half 1 of the layer may overwrite the accumulator
    } else {
        // every MMA of layer l is complete: its operand is dead, the next one goes over it.  The held half goes first
        t2_store(a_lo, nch, hold);
        tmem_st_wait();
        tc_fence_before();
        arrive(S_A_FULL);
        T2_READ_CONVERT(acc0, hold);
        tc_fence_before();
        arrive(S_DH_FREE);
        t2_store(a_hi, nch, hold);
        tmem_st_wait();
        tc_fence_before();
        arrive(S_A_FULL + 1);
    }
#undef T2_READ_CONVERT
#undef T2_PAIR
}

template <int CG, int ACT, bool F16>
__global__ void __launch_bounds__(T2_THREADS, 1)
hb_sur_tc2_kernel(HbParticles p, size_t n, const __grid_constant__ HbSurDev sd, const __grid_constant__ T2Plan pl,
                  double* __restrict__ partials) {
    constexpr int PROD_WARP = 12, MMA_WARP = 13;          // MMA warps: 13 (slot 0), 14 (slot 1)
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    // the 128-byte swizzle atoms (8 rows x 128 B) must sit on 1024-byte boundaries of the shared window
    unsigned char* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    const uint32_t sbase = smem_u32(smem);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const uint32_t rank = CG == 1 ? 0u : cluster_rank();
    const size_t ntiles = (n + TILE_M - 1) / TILE_M;
    const size_t ngroups = (ntiles + CG - 1) / CG;
    const size_t cluster_id = blockIdx.x / CG, nclusters = gridDim.x / CG;
    // tile groups of this CTA (pair): g_k = cluster_id + k * nclusters, k < nk; slot = k & 1, use count it = k >> 1
    const uint32_t nk = cluster_id < ngroups ? (uint32_t)((ngroups - cluster_id + nclusters - 1) / nclusters) : 0u;
    const int L = pl.n_linear;
    const int P = 2 * (L - 2) + 2;             // phases per tile: a, (1,0), (1,1), ..., (L-2,1), d

    const uint32_t bar0 = sbase + pl.bar_off;
    auto bar = [&](int i) -> uint32_t { return bar0 + 8u * (uint32_t)i; };
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + pl.bar_off + 8 * T_COUNT);
    float* bias_s = reinterpret_cast<float*>(smem + pl.bias_base);

    if (tid == 0) {
        mbar_init(bar(T_W), 1);
        for (int s = 0; s < T2_STAGES; ++s) {
            mbar_init(bar(T_IN_FULL + s), 1);
            mbar_init(bar(T_IN_EMPTY + s), 4);
        }
        for (int t = 0; t < 2; ++t) {
            const int b = T_SLOT + 8 * t;
            mbar_init(bar(b + S_A0_FULL), 4 * CG);
            mbar_init(bar(b + S_A0_FULL + 1), 4 * CG);
            mbar_init(bar(b + S_DH_FULL), 1);
            mbar_init(bar(b + S_DH_FREE), 4 * CG);
            mbar_init(bar(b + S_A_FULL), 4 * CG);
            mbar_init(bar(b + S_A_FULL + 1), 4 * CG);
            mbar_init(bar(b + S_D_LAST), 1);
            mbar_init(bar(b + S_OUT_READ), 4 * CG);
        }
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
            for (uint32_t k = 0; k < nk; ++k) {
                const size_t tile = (cluster_id + (size_t)k * nclusters) * CG + rank;
                const bool full = tile < ntiles && (tile + 1) * TILE_M <= n;
                if (full) {
                    mbar_wait<false>(bar(T_IN_EMPTY + stage), ph ^ 1);
                    mbar_expect_tx(bar(T_IN_FULL + stage), STAGE_BYTES);
                    for (int j = 0; j < 6; ++j)
                        bulk_g2s(sbase + pl.stage_off + stage * STAGE_BYTES + j * TILE_M * 4, p.v[j] + tile * TILE_M,
                                 TILE_M * 4, bar(T_IN_FULL + stage));
                    if (++stage == T2_STAGES) { stage = 0; ph ^= 1; }
                }
            }
        }
        __syncwarp();
    } else if (warp >= MMA_WARP) {
        // ===================================================== MMA issuer of slot T (leader CTA of the pair only)
        // The whole warp walks its slot's phases (warp-uniform control flow, barrier waits by every lane); one elected
        // lane issues the MMAs and commits (tcgen05.commit tracks the MMAs of the thread that executes it: per slot).
        if (rank == 0) {
            const uint32_t T = (uint32_t)(warp - MMA_WARP);
            const uint32_t fmt = F16 ? 0u : 1u;
            const uint32_t idesc_base = (1u << 4) | (fmt << 7) | (fmt << 10) | ((uint32_t)((TILE_M * CG) >> 4) << 24);
            const bool issuer = elect_one();
            const uint64_t w0_desc = make_desc_l0(sbase + pl.w_off[0]);
            const uint32_t n_it = T == 0 ? (nk + 1) / 2 : nk / 2;
            const uint32_t sb = tmem_base + T * T2_SLOT_COLS;
            const uint32_t d_tmem = sb + T2_DH;
            const int sbar = T_SLOT + 8 * (int)T;
            uint32_t ph_free = 0, ph_a = 0;        // ph_free; bit kh of ph_a: parity of the next completion
            for (uint32_t it = 0; it < n_it; ++it) {
                const uint64_t a0d = make_desc_l0(sbase + pl.a0_off + (2 * T + (it & 1)) * A0_BYTES);
                // phase a.  The slot's columns still hold the previous tile's outputs until the IO warps read them.
                if (it > 0) mbar_wait<true>(bar(sbar + S_OUT_READ), (it - 1) & 1);
                mbar_wait<true>(bar(sbar + S_A0_FULL + (int)(it & 1)), (it >> 1) & 1);
                tc_fence_after();
                if (issuer) {
                    umma<CG, false>(sb, a0d, w0_desc, idesc_base | ((uint32_t)(pl.npad[0] >> 3) << 17));
                    umma_commit<CG>(bar(sbar + S_DH_FULL));
                }
                __syncwarp();
                for (int ph = 1; ph < P; ++ph) {
                    const bool last = ph == P - 1;
                    const int l = last ? L - 1 : 1 + ((ph - 1) >> 1);
                    const int h = last ? 0 : ((ph - 1) & 1);
                    const uint32_t idesc = idesc_base | ((uint32_t)(pl.hw[l] >> 3) << 17);
                    const int ksteps = pl.npad[l - 1] >> 4, kb = pl.npad[l - 1] >> 5;   // K = 16 steps; first step of K-half 1
                    const uint32_t half_rows = (uint32_t)(h * (pl.hw[l] / CG));
                    const uint64_t bd = make_desc(sbase + pl.w_off[l] + half_rows * 128u);
                    const uint64_t bd_step = (uint64_t)(pl.w_slab_bytes[l] >> 4);
                    const uint64_t wbd = make_desc_l0(sbase + pl.wb_off[l] + half_rows * 32u);
                    // the accumulator columns: read by the epilogue warps (previous phase of this slot)
                    mbar_wait<true>(bar(sbar + S_DH_FREE), ph_free);
                    ph_free ^= 1u;
                    tc_fence_after();
                    // hidden layer: the bias goes in first, as one K = 16 MMA of the tile's layer-0 operand (ones in
                    // columns 12, 13) with this half's bias block (b_hi, b_lo in columns 12, 13, zeros elsewhere)
                    if (!last && issuer) umma<CG, false>(d_tmem, a0d, wbd, idesc);
                    const bool fresh = h == 0;      // the operand was written since the last phase: wait per K-half
                    bool seen1 = false;
                    for (int k0 = 0; k0 < ksteps; k0 += 4) {
                        if (fresh && k0 == 0) {
                            mbar_wait<true>(bar(sbar + S_A_FULL), ph_a & 1);
                            ph_a ^= 1u;
                            tc_fence_after();
                        }
                        if (fresh && !seen1 && k0 + 4 > kb) {      // this slab reaches into K-half 1
                            mbar_wait<true>(bar(sbar + S_A_FULL + 1), (ph_a >> 1) & 1);
                            ph_a ^= 2u;
                            tc_fence_after();
                            seen1 = true;
                        }
                        if (issuer) {
                            // one 64-wide K slab: four K = 16 steps, B advances by 32 B, A by 8 columns
                            const uint32_t ad = sb + (uint32_t)(8 * k0);
                            const uint64_t bj = bd + (uint64_t)(k0 >> 2) * bd_step;
                            if (k0 == 0 && last) umma_ts<CG, false>(d_tmem, ad, bj, idesc);
                            else umma_ts<CG, true>(d_tmem, ad, bj, idesc);
                            umma_ts<CG, true>(d_tmem, ad + 8, bj + 2, idesc);
                            umma_ts<CG, true>(d_tmem, ad + 16, bj + 4, idesc);
                            umma_ts<CG, true>(d_tmem, ad + 24, bj + 6, idesc);
                        }
                    }
                    if (issuer) umma_commit<CG>(bar(sbar + (last ? S_D_LAST : S_DH_FULL)));
                    __syncwarp();
                }
            }
        }
        __syncwarp();
    } else if (warp < EPI_WARP0) {
        // ===================================================== IO warps: prologue of tile k + 2, output of tile k
        const int wq = warp & 3;                 // TMEM lane quarter this warp may access
        const int row = 32 * wq + lane;          // tile row = TMEM lane = particle within the tile
        const uint32_t a0_row = sbase + pl.a0_off + (uint32_t)(row >> 3) * 256 + (uint32_t)(row & 7) * 16;
        const uint32_t tlane = tmem_base + ((uint32_t)(32 * wq) << 16) + T2_DH;
        const float* bl = bias_s;
        HbMomAcc acc;
        acc.clear();
        int stage = 0;
        uint32_t pin = 0;
        // a4: load, convert, normalise, split, write the layer-0 operand of tile group k
        auto prologue = [&](uint32_t k) {
            const size_t tile = (cluster_id + (size_t)k * nclusters) * CG + rank;
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
                if (++stage == T2_STAGES) { stage = 0; pin ^= 1; }
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
            const uint32_t T = k & 1u, buf = (k >> 1) & 1u;
            const uint32_t dst = a0_row + (2 * T + buf) * A0_BYTES;
            sts128(dst, q0);
            sts128(dst + 128, q1);
            fence_proxy_async();
            __syncwarp();
            if (lane == 0) mbar_arrive_cluster(bar(T_SLOT + 8 * (int)T + S_A0_FULL + (int)buf), 0);
        };
        mbar_wait<false>(bar(T_W), 0);           // this CTA's weights are resident before the first MMA may start
        if (nk > 0) prologue(0);
        if (nk > 1) prologue(1);
        for (uint32_t k = 0; k < nk; ++k) {
            // buffer (k >> 1) + 1 & 1 of the slot was last read by tile k - 2, whose output was taken two turns ago
            if (k + 2 < nk) prologue(k + 2);
            const uint32_t T = k & 1u, it = k >> 1;
            const size_t tile = (cluster_id + (size_t)k * nclusters) * CG + rank;
            const size_t i = tile * TILE_M + row;
            const bool valid = tile < ntiles && i < n;
            mbar_wait<false>(bar(T_SLOT + 8 * (int)T + S_D_LAST), it & 1);
            tc_fence_after();
            uint32_t r[8];
            tmem_ld8(tlane + T * T2_SLOT_COLS, r);
            tmem_ld_wait();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive_cluster(bar(T_SLOT + 8 * (int)T + S_OUT_READ), 0);
            if (valid) {
                float w[6];
#pragma unroll
                for (int j = 0; j < 6; ++j) w[j] = __uint_as_float(r[j]) + bl[j];
                float x, px, y, py, t, pt;
                hb_sur_epilogue(sd, w, x, px, y, py, t, pt);
                p.v[0][i] = x; p.v[1][i] = px; p.v[2][i] = y; p.v[3][i] = py; p.v[4][i] = t; p.v[5][i] = pt;
                if (partials) acc.add(sd.mom_pivot, x, px, y, py, t, pt);
            }
        }
        if (partials) {
            double* red = reinterpret_cast<double*>(smem + pl.red_off);
            hb_block_reduce_moments(acc, red, partials + blockIdx.x, tid - 32 * IO_WARP0, 128, 2);
        }
    } else {
        // ===================================================== hidden-layer epilogue warps of slot T
        const int wq = warp & 3;
        const uint32_t T = (uint32_t)((warp - EPI_WARP0) >> 2);
        const uint32_t tl = tmem_base + ((uint32_t)(32 * wq) << 16) + T * T2_SLOT_COLS;
        const uint32_t sbar0 = bar0 + 8u * (uint32_t)(T_SLOT + 8 * (int)T);
        const uint32_t n_it = T == 0 ? (nk + 1) / 2 : nk / 2;
        uint32_t par = 0;                         // parity of the next completion of DH_FULL
        uint32_t hold[64];                        // packed half 0 of the layer in flight
        for (uint32_t it = 0; it < n_it; ++it)
            for (int ph = 0; ph < P - 1; ++ph) {  // phase d belongs to the IO warps
                t2_epilogue_phase<ACT, F16>(sd, pl, sbar0, tl, ph, par, lane, hold);
                par ^= 1u;
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
        pl.hw[l] = (l == 0 || last) ? pl.npad[l] : pl.npad[l] / 2;
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
    off += 4 * A0_BYTES;
    pl.stage_off = off;
    off += T2_STAGES * STAGE_BYTES;
    pl.bias_base = off;
    off += t2_round_up(pl.npad[n_linear - 1] * 4, 16);
    pl.bar_off = off;
    off += t2_round_up(8 * T_COUNT + 8, 16);
    pl.red_off = off;
    off += 4 * HB_NMOM * 8;
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
//   layer 0 (K = 16, no swizzle): per 8-row group 256 bytes = K chunk 0 of the 8 rows (8 x 16 B), then K chunk 1; W_0 is
//     carried twice (columns 0..5 meet the hi parts of the inputs, 6..11 the lo parts), b_hi, b_lo in columns 12, 13;
//     rank r holds the rows of neurons [r npad/cg, (r+1) npad/cg).
//   hidden layer l: per 64-wide K slab, per rank npad/cg rows of 128 bytes (K-major, 128-byte swizzle: the 16-byte chunk
//     c of local row i sits at chunk position c ^ (i mod 8)); local row h (hw/cg) + i of rank r is neuron
//     h hw + r (hw/cg) + i: the rows of N-half 0 first, then those of N-half 1 (a cta_group::2 MMA of N = hw takes hw/2
//     rows from each CTA).  Behind the slabs the bias block (K = 16 operand as layer 0, same row order).
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
