// hb_sur_tc.cu -- surrogate stage on the 5th-gen tensor cores (HB_PREC_BF16 / HB_PREC_F16): rows a4-a6.
//
// One 128-particle tile per CTA (one TMEM lane per particle; a CTA pair works on 256 particles with
// cta_group::2).  Warp roles:
//   warp 4+4G   copy producer : weights once, then the six coordinate rows of each tile through the TMA
//                               engine (cp.async.bulk + mbarrier complete_tx) into a 2-stage ring.
//   warp 5+4G   MMA issuer    : one elected thread (leader CTA of a pair) issues every tcgen05.mma.
//   warps 0-3   IO warps      : a4 prologue (s->t R6 in deviation form, normalise R8, hi/lo split, layer-0
//                               operand) of tile i+1, then a6 epilogue of tile i (tcgen05.ld of the 6 outputs,
//                               de-normalise R8, reference update R7, t->s R6, coalesced store, fp64 moments R10).
//   warps 4..   4G hidden-layer epilogue warps: tcgen05.ld of 32 accumulator columns (bias already inside, see
//                               below), sigma (Eq. 1/2, tanh), round to 16 bit, tcgen05.st of the 16 packed columns
//                               over the first half of the columns just read.  Hidden activations never leave
//                               tensor memory (they never touch HBM).
// Bias.  The layer-0 operand row is  hi0..5, lo0..5, 1, 1, 0, 0;  W_0 carries b_hi, b_lo (bias rounded to the
// operand type + rounded remainder) in K columns 12, 13.  Every hidden layer gets one extra K = 16 MMA of that same
// operand tile against a bias block (b_hi, b_lo in columns 12, 13, zeros elsewhere) with accumulate = 0, issued
// before the layer's first K slab is awaited.
// Operand.  Layer l >= 1 reads A from tensor memory (tcgen05.mma [d], [a], b-desc): K step kappa of slab j is the
// 8 columns at 64 j + 32 (kappa / 2) + 8 (kappa mod 2) of D[(l-1) & 1]; shared memory only feeds B.
// Pipeline.  The accumulator is double-buffered in TMEM.  The hidden-layer accumulators of a CTA form one sequence of
// EVENTS e = 0, 1, 2, ... (tile t, layer l < L-1: e = t (L-1) + l); event e lives in D[e & 1], signals D_HID[e & 1] and
// its operand slabs SLAB_FULL[e & 1][j].  The next operand is handed to the MMA issuer per 64-column K slab: the MMAs
// of layer l+1 start as soon as the epilogue of layer l has converted slab 0 and then run back to back while the
// epilogue finishes the other slabs.  The last layer (N = 16) does not take a buffer of its own: it writes its 16
// output columns into the gap [16,32) that the in-place packing leaves in chunk 0 of its operand's buffer.  The
// other buffer is dead by then (it held the operand of layer L-2), so layer 0 of the NEXT tile is issued into it
// right behind layer L-2 of the current one: its epilogue runs under the current tile's last layer and output, and
// the tensor pipe does not wait for it (one of the four hand-overs per tile of a 6-256^3-6 net is gone).
#include "hb_tc_common.cuh"

namespace {

struct TcPlan {
    int n_linear;
    int ksteps[HB_MAX_LINEAR];        // K = 16 MMA steps of layer l
    int nslab[HB_MAX_LINEAR];         // 64-wide K slabs of layer l's operands (layer 0: 0, compact layout)
    int npad[HB_MAX_LINEAR];          // padded fan-out (whole layer, both CTAs of a pair)
    int w_off[HB_MAX_LINEAR];         // smem byte offset of layer l's weights (this CTA's rows)
    int w_slab_bytes[HB_MAX_LINEAR];  // l >= 1: (npad / CG) * 128;  l = 0: (npad / CG) * 32 (whole layer)
    int wb_off[HB_MAX_LINEAR];        // 1 <= l <= L-2: smem byte offset of layer l's bias block (K = 16 operand, this CTA's rows)
    int wb_bytes[HB_MAX_LINEAR];      //                (npad / CG) * 32
    int a0_off, stage_off, bias_base, bar_off, red_off, total;
    int d_cols;                       // columns of one accumulator buffer
    int tmem_cols;                    // 2 * d_cols rounded to a power of two >= 32
    int w_bytes_total;                // bytes this CTA loads
};

// ------------------------------------------------------------------------------- kernel
// barrier block (8 bytes each, at pl.bar_off):
enum : int {
    B_W = 0,              // weights resident (local)
    B_IN_FULL = 1,        // [2] coordinate rows staged (local)
    B_IN_EMPTY = 3,       // [2] stage consumed by the 4 IO warps (local)
    B_A0_FULL = 5,        // [2] layer-0 operand written (leader; 4 IO warps x CG)
    B_SLAB_FULL = 7,      // [2][MAX_SLABS] K slab of the operand packed from event e, set e & 1 (leader; 4G warps x CG)
    B_D_HID = 15,         // [2] accumulator D[e & 1] of hidden event e complete (both CTAs, MMA commit)
    B_D_LAST = 17,        // accumulator of the last layer complete (both CTAs, MMA commit)
    B_OUT_READ = 18,      // last layer's accumulator read by the IO warps (leader; 4 IO warps x CG)
    B_COUNT = 19
};

template <int CG, int ACT, bool F16, int G>
__global__ void __launch_bounds__(tc_threads(G), G == 1 ? 2 : 1)
hb_sur_tc_kernel(HbParticles p, size_t n, const __grid_constant__ HbSurDev sd, const __grid_constant__ TcPlan pl,
                 double* __restrict__ partials) {
    constexpr int THREADS = tc_threads(G);
    // the scheduler favours the highest warp id: the MMA issuer sits on top so that busy epilogue warps on the
    // same scheduler never delay an MMA issue
    constexpr int PROD_WARP = EPI_WARP0 + 4 * G, MMA_WARP = PROD_WARP + 1;
    static_assert(G == 1 || G == 2, "epilogue warps = 4 x G");
    constexpr int CW = 32;                           // accumulator columns per epilogue step of one warp
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    // the 128-byte swizzle atoms (8 rows x 128 B) must sit on 1024-byte boundaries of the shared window
    unsigned char* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    const uint32_t sbase = smem_u32(smem);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const uint32_t rank = CG == 1 ? 0u : cluster_rank();
    const size_t ntiles = (n + TILE_M - 1) / TILE_M;
    const size_t ngroups = (ntiles + CG - 1) / CG;
    const size_t cluster_id = blockIdx.x / CG, nclusters = gridDim.x / CG;
    const int L = pl.n_linear;
    constexpr uint32_t OUT_GAP = 16;          // L >= 2: the 16 output columns sit in the gap of chunk 0 of the operand's buffer

    const uint32_t bar0 = sbase + pl.bar_off;
    auto bar = [&](int i) -> uint32_t { return bar0 + 8u * (uint32_t)i; };
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + pl.bar_off + 8 * B_COUNT);
    float* bias_s = reinterpret_cast<float*>(smem + pl.bias_base);

    if (tid == 0) {
        mbar_init(bar(B_W), 1);
        for (int s = 0; s < IN_STAGES; ++s) {
            mbar_init(bar(B_IN_FULL + s), 1);
            mbar_init(bar(B_IN_EMPTY + s), 4);
            mbar_init(bar(B_A0_FULL + s), 4 * CG);
            mbar_init(bar(B_D_HID + s), 1);
        }
        for (int j = 0; j < 2 * MAX_SLABS; ++j) mbar_init(bar(B_SLAB_FULL + j), 4 * G * CG);
        mbar_init(bar(B_D_LAST), 1);
        mbar_init(bar(B_OUT_READ), 4 * CG);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == MMA_WARP) {
        tmem_alloc<CG>(smem_u32(tmem_slot), (uint32_t)pl.tmem_cols);
        tmem_relinquish<CG>();
    }
    // bias of the last layer -> shared (fp32, added by the IO warps); the hidden layers' biases ride in the MMAs
    for (int i = tid; i < pl.npad[L - 1]; i += THREADS) bias_s[i] = sd.btc[sd.btc_off[L - 1] + i];
    tc_fence_before();
    __syncthreads();
    if (CG == 2) cluster_sync_all();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    if (warp == PROD_WARP) {
        // ===================================================== producer: weights once, then particle tiles
        if (lane == 0) {
            mbar_expect_tx(bar(B_W), (uint32_t)pl.w_bytes_total);
            const unsigned char* wg = reinterpret_cast<const unsigned char*>(sd.wtc);
            // layer 0: one contiguous block of this CTA's rows
            bulk_g2s(sbase + pl.w_off[0], wg + sd.wtc_off[0] + (size_t)rank * pl.w_slab_bytes[0],
                     (uint32_t)pl.w_slab_bytes[0], bar(B_W));
            for (int l = 1; l < L; ++l)
                for (int s = 0; s < pl.nslab[l]; ++s) {
                    const unsigned char* src = wg + sd.wtc_off[l] + (size_t)s * pl.npad[l] * 128 + (size_t)rank * pl.w_slab_bytes[l];
                    bulk_g2s(sbase + pl.w_off[l] + s * pl.w_slab_bytes[l], src, (uint32_t)pl.w_slab_bytes[l], bar(B_W));
                }
            for (int l = 1; l + 1 < L; ++l)      // bias blocks of the hidden layers (behind the layer's K slabs)
                bulk_g2s(sbase + pl.wb_off[l],
                         wg + sd.wtc_off[l] + (size_t)pl.nslab[l] * pl.npad[l] * 128 + (size_t)rank * pl.wb_bytes[l],
                         (uint32_t)pl.wb_bytes[l], bar(B_W));
            int stage = 0;
            uint32_t ph = 0;
            for (size_t g = cluster_id; g < ngroups; g += nclusters) {
                const size_t tile = g * CG + rank;
                const bool full = tile < ntiles && (tile + 1) * TILE_M <= n;
                if (full) {
                    mbar_wait<false>(bar(B_IN_EMPTY + stage), ph ^ 1);
                    mbar_expect_tx(bar(B_IN_FULL + stage), STAGE_BYTES);
                    for (int j = 0; j < 6; ++j)
                        bulk_g2s(sbase + pl.stage_off + stage * STAGE_BYTES + j * TILE_M * 4, p.v[j] + tile * TILE_M,
                                 TILE_M * 4, bar(B_IN_FULL + stage));
                    stage ^= 1;
                    if (stage == 0) ph ^= 1;
                }
            }
        }
        __syncwarp();
    } else if (warp == MMA_WARP) {
        // ===================================================== MMA issuer (leader CTA of the pair only)
        // The whole warp walks the schedule (warp-uniform control flow, barrier waits by every lane); one
        // elected lane issues the MMAs and commits.
        if (rank == 0) {
            const uint32_t fmt = F16 ? 0u : 1u;
            const uint32_t idesc_base = (1u << 4) | (fmt << 7) | (fmt << 10) | ((uint32_t)((TILE_M * CG) >> 4) << 24);
            const bool issuer = elect_one();
            const uint64_t w0_desc = make_desc_l0(sbase + pl.w_off[0]);
            uint32_t ph_slab = 0;                    // bit 4 set + j: parity of the next completion of SLAB_FULL[set][j]
            // per-layer constants are fetched one layer ahead: anything issued behind a batch of MMAs waits for
            // the tensor pipe, so the loads for layer l+1 go out before the MMAs of layer l
            struct LayerC { uint32_t idesc; int nsl; uint64_t bd, bd_step, wbd; };
            auto layer_consts = [&](int l) {
                LayerC c;
                c.idesc = idesc_base | ((uint32_t)(pl.npad[l] >> 3) << 17);
                c.nsl = pl.nslab[l];
                c.bd = make_desc(sbase + pl.w_off[l]);
                c.bd_step = (uint64_t)(pl.w_slab_bytes[l] >> 4);
                c.wbd = make_desc_l0(sbase + pl.wb_off[l]);
                return c;
            };
            const LayerC c0 = layer_consts(0);
            const bool more_than_one = L > 1;
            const uint32_t nmine = cluster_id < ngroups ? (uint32_t)((ngroups - cluster_id + nclusters - 1) / nclusters) : 0u;
            // out_in[x]: 1 + the tile whose 16 output columns sit in D[x] and may not have been read yet (0: none).
            // Whatever overwrites D[x] as a whole (layer 0, a hidden layer's bias MMA) waits for the IO warps first.
            uint32_t out_in0 = 0u, out_in1 = 0u;
            auto claim = [&](uint32_t x) {
                const uint32_t v = x ? out_in1 : out_in0;
                if (v) {
                    mbar_spin(bar(B_OUT_READ), (v - 1) & 1);
                    if (x) out_in1 = 0u; else out_in0 = 0u;
                }
            };
            // layer 0 of tile `t` = hidden event e0 = t (L-1) (or the tile's output when L = 1): one K = 16 MMA from the
            // compact operand buffers into D[e0 & 1]
            auto issue_l0 = [&](uint32_t t) {
                const uint32_t x = more_than_one ? ((t * (uint32_t)(L - 1)) & 1u) : 0u;
                claim(x);
                mbar_spin(bar(B_A0_FULL + (t & 1)), (t >> 1) & 1);
                tc_fence_after();
                if (issuer) {
                    umma<CG, false>(tmem_base + x * (uint32_t)pl.d_cols, make_desc_l0(sbase + pl.a0_off + (t & 1) * A0_BYTES),
                                    w0_desc, c0.idesc);
                    umma_commit<CG>(more_than_one ? bar(B_D_HID + (int)x) : bar(B_D_LAST));
                }
                __syncwarp();
                if (!more_than_one) out_in0 = t + 1;
            };
            if (nmine > 0) issue_l0(0);
            if (L == 2 && nmine > 1) issue_l0(1);        // layer L-2 IS layer 0: the next tile's goes out right behind it
            LayerC nxt = layer_consts(more_than_one ? 1 : 0);
            for (uint32_t it = 0; it < nmine; ++it) {
                for (int l = 1; l < L; ++l) {
                    const LayerC cur = nxt;
                    nxt = layer_consts(l + 1 < L ? l + 1 : 1);
                    const bool hid = l + 1 < L;
                    // layer l consumes hidden event e_in (operand packed in place in D[e_in & 1]: slab j = columns
                    // [64 j, 64 j + 16) and [64 j + 32, 64 j + 48), 8 per K = 16 step); a hidden layer produces event
                    // e_in + 1 in the other buffer, the last layer writes the gap of its operand's buffer
                    const uint32_t e_in = it * (uint32_t)(L - 1) + (uint32_t)(l - 1);
                    const uint32_t xin = e_in & 1u, xout = hid ? xin ^ 1u : xin;
                    const uint32_t a_tmem = tmem_base + xin * (uint32_t)pl.d_cols;
                    const uint32_t d_tmem = tmem_base + xout * (uint32_t)pl.d_cols + (hid ? 0u : OUT_GAP);
                    const uint32_t idesc = cur.idesc;
                    const int nsl = cur.nsl;
                    const uint64_t bd = cur.bd, bd_step = cur.bd_step;
                    if (hid) claim(xout);
                    // hidden layer: the bias goes in first, as one K = 16 MMA of this tile's layer-0 operand (ones
                    // in columns 12, 13) with the layer's bias block (b_hi, b_lo in columns 12, 13, zeros elsewhere).
                    // It depends on nothing the epilogue produces, so it runs in the bubble before slab 0 arrives.
                    if (hid && issuer)
                        umma<CG, false>(d_tmem, make_desc_l0(sbase + pl.a0_off + (it & 1) * A0_BYTES), cur.wbd, idesc);
                    // The K slabs of the operand arrive one by one from the epilogue warps.  One probe first: lane j
                    // tests slab j's barrier (test_wait does not suspend) and a ballot tells the warp how many leading
                    // slabs are already there -- for the last layer, whose operand is usually complete, that is one
                    // ~150-cycle probe instead of four (polled one by one, the probes cost more than its 16 small MMAs
                    // take).  The slabs that are not there yet are awaited one by one (try_wait sleeps in hardware and
                    // wakes ~60 cycles after the last arrive).
                    const int sset = (int)xin * MAX_SLABS;
                    const int my_slab = lane < MAX_SLABS ? lane : 0;
                    const uint32_t ok = lane < nsl ? mbar_test(bar(B_SLAB_FULL + sset + my_slab), (ph_slab >> (sset + my_slab)) & 1u) : 0u;
                    const uint32_t have = __ballot_sync(0xffffffffu, ok != 0u);
                    int there = 0;
                    while (there < nsl && ((have >> there) & 1u)) ++there;
                    if (there > 0) tc_fence_after();
#pragma unroll
                    for (int j = 0; j < MAX_SLABS; ++j) {
                        if (j < nsl) {
                            if (j >= there) {
                                mbar_spin(bar(B_SLAB_FULL + sset + j), (ph_slab >> (sset + j)) & 1);
                                tc_fence_after();
                            }
                            if (issuer) {
                                // four K = 16 steps inside the 64-wide slab: B advances by 32 B, A by 8 columns
                                // (second 32-column chunk of the slab: + 32)
                                const uint32_t ad = a_tmem + (uint32_t)(64 * j);
                                const uint64_t bj = bd + (uint64_t)j * bd_step;
                                if (j == 0 && !hid) umma_ts<CG, false>(d_tmem, ad, bj, idesc);
                                else umma_ts<CG, true>(d_tmem, ad, bj, idesc);
                                umma_ts<CG, true>(d_tmem, ad + 8, bj + 2, idesc);
                                umma_ts<CG, true>(d_tmem, ad + 32, bj + 4, idesc);
                                umma_ts<CG, true>(d_tmem, ad + 40, bj + 6, idesc);
                            }
                        }
                    }
                    ph_slab ^= ((1u << nsl) - 1u) << sset;
                    if (issuer) umma_commit<CG>(hid ? bar(B_D_HID + (int)xout) : bar(B_D_LAST));
                    __syncwarp();
                    if (!hid) { if (xout) out_in1 = it + 1; else out_in0 = it + 1; }
                    // behind layer L-2 the buffer that held its operand is dead: layer 0 of the next tile goes there
                    // (for L = 2 that was done one tile ahead; keep one tile ahead)
                    if (L > 2 && l == L - 2 && it + 1 < nmine) issue_l0(it + 1);
                }
                if (L == 2 && it + 2 < nmine) issue_l0(it + 2);
                if (L == 1 && it + 1 < nmine) issue_l0(it + 1);
            }
        }
        __syncwarp();
    } else if (warp < EPI_WARP0) {
        // ===================================================== IO warps: prologue of tile i+1, output of tile i
        const int wq = warp & 3;                 // TMEM lane quarter this warp may access
        const int row = 32 * wq + lane;          // tile row = TMEM lane = particle within the tile
        const uint32_t a0_row = sbase + pl.a0_off + (uint32_t)(row >> 3) * 256 + (uint32_t)(row & 7) * 16;
        const uint32_t tlane = tmem_base + ((uint32_t)(32 * wq) << 16);
        const float* bl = bias_s;
        HbMomAcc acc;
        acc.clear();
        int stage = 0;
        uint32_t pin = 0;
        // a4: load, convert, normalise, split, write the layer-0 operand of the tile of group g
        auto prologue = [&](size_t g, uint32_t buf) {
            const size_t tile = g * CG + rank;
            const size_t i = tile * TILE_M + row;
            const bool valid = tile < ntiles && i < n;
            const bool full = tile < ntiles && (tile + 1) * TILE_M <= n;
            float c[6] = {0, 0, 0, 0, 0, 0};
            if (full) {
                mbar_wait<false>(bar(B_IN_FULL + stage), pin);
                const float* st = reinterpret_cast<const float*>(smem + pl.stage_off + stage * STAGE_BYTES);
#pragma unroll
                for (int j = 0; j < 6; ++j) c[j] = st[j * TILE_M + row];
                __syncwarp();
                if (lane == 0) mbar_arrive_local(bar(B_IN_EMPTY + stage));
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
            const uint32_t dst = a0_row + buf * A0_BYTES;
            asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(dst), "r"(q0[0]), "r"(q0[1]), "r"(q0[2]), "r"(q0[3]) : "memory");
            asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(dst + 128), "r"(q1[0]), "r"(q1[1]), "r"(q1[2]), "r"(q1[3]) : "memory");
            fence_proxy_async();
            __syncwarp();
            if (lane == 0) mbar_arrive_cluster(bar(B_A0_FULL + buf), 0);
        };
        mbar_wait<false>(bar(B_W), 0);           // this CTA's weights are resident before the first MMA may start
        uint32_t it = 0;
        if (cluster_id < ngroups) prologue(cluster_id, 0);
        for (size_t g = cluster_id; g < ngroups; g += nclusters, ++it) {
            if (g + nclusters < ngroups) prologue(g + nclusters, (it + 1) & 1);
            const size_t tile = g * CG + rank;
            const size_t i = tile * TILE_M + row;
            const bool valid = tile < ntiles && i < n;
            mbar_wait<false>(bar(B_D_LAST), it & 1);
            tc_fence_after();
            uint32_t r[8];
            // the outputs sit in the gap of the buffer of the tile's last hidden event (L = 1: at column 0 of D[0])
            const uint32_t e_last = it * (uint32_t)(L - 1) + (uint32_t)(L - 2);
            tmem_ld8(L > 1 ? tlane + (e_last & 1u) * (uint32_t)pl.d_cols + OUT_GAP : tlane, r);
            tmem_ld_wait();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive_cluster(bar(B_OUT_READ), 0);
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
        // ===================================================== hidden-layer epilogue warps
        const int wq = warp & 3;
        const int grp = (warp - EPI_WARP0) >> 2;  // column group inside every 64-column slab
        const uint32_t tlane = tmem_base + ((uint32_t)(32 * wq) << 16);
        uint32_t ph_d = 0;                        // bit b: parity of the next completion of D_HID[b]
        const uint32_t nmine = cluster_id < ngroups ? (uint32_t)((ngroups - cluster_id + nclusters - 1) / nclusters) : 0u;
        const uint32_t nev = nmine * (uint32_t)(L - 1);        // hidden events of this CTA, in the order they are issued
        int l = 0;
        for (uint32_t e = 0; e < nev; ++e) {
            const int b = (int)(e & 1u);
            const int nsl = pl.npad[l] >> 6;
            const float slope = sd.prelu[l];
            // this warp's 32-column chunks of the layer: columns 32 * (c * G + grp), c = 0 .. nch-1
            // (G = 2: one chunk per 64-column slab; G = 1: both chunks of every slab)
            const int nch = nsl * (2 / G);
            const uint32_t tl = tlane + (uint32_t)(b * pl.d_cols);
            const int sset = B_SLAB_FULL + b * MAX_SLABS;
            mbar_wait<true>(bar(B_D_HID + b), (ph_d >> b) & 1);
            ph_d ^= 1u << b;
            tc_fence_after();
            uint32_t ra[CW], rb[CW];
            tmem_ld<CW>(tl + (uint32_t)(grp * CW), ra);
            for (int c = 0; c < nch; c += 2) {
                const int col_a = CW * (c * G + grp), col_b = CW * ((c + 1) * G + grp);
                tmem_ld_wait();
                if (c + 1 < nch) tmem_ld<CW>(tl + (uint32_t)col_b, rb);
                epi_store_tmem<ACT, F16>(ra, tl + (uint32_t)col_a, slope);
                if (G == 2 || c + 1 >= nch) {           // chunk a closes its slab
                    tmem_st_wait();
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) mbar_arrive_cluster(bar(sset + (col_a >> 6)), 0);
                }
                if (c + 1 < nch) {
                    tmem_ld_wait();
                    if (c + 2 < nch) tmem_ld<CW>(tl + (uint32_t)(CW * ((c + 2) * G + grp)), ra);
                    epi_store_tmem<ACT, F16>(rb, tl + (uint32_t)col_b, slope);
                    tmem_st_wait();
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) mbar_arrive_cluster(bar(sset + (col_b >> 6)), 0);
                }
            }
            if (++l == L - 1) l = 0;
        }
    }
    // ---- teardown: everyone done with TMEM (both CTAs of a pair), then free it
    tc_fence_before();
    __syncthreads();
    if (CG == 2) cluster_sync_all();
    if (warp == MMA_WARP) {
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
        if (l == 0) { kpad[l] = 16; ksteps[l] = 1; }                 // 6 hi + 6 lo + 4 zero
        else { kpad[l] = npad[l - 1]; ksteps[l] = npad[l - 1] / 16; }
    }
}

bool make_plan(int cg, int n_linear, const int* widths, TcPlan& pl) {
    std::memset(&pl, 0, sizeof pl);
    int kpad[HB_MAX_LINEAR], ksteps[HB_MAX_LINEAR];
    layer_geometry(n_linear, widths, kpad, pl.npad, ksteps);
    pl.n_linear = n_linear;
    int off = 0, maxslab = 1, maxn = 32;
    for (int l = 0; l < n_linear; ++l) {
        pl.ksteps[l] = ksteps[l];
        pl.nslab[l] = l == 0 ? 0 : kpad[l] / 64;
        if ((pl.npad[l] / cg) % 8) return false;
        pl.w_slab_bytes[l] = pl.npad[l] / cg * (l == 0 ? 32 : 128);
        pl.w_off[l] = off;
        off += (l == 0 ? 1 : pl.nslab[l]) * pl.w_slab_bytes[l];
        if (l >= 1 && l + 1 < n_linear) {
            pl.wb_off[l] = off;
            pl.wb_bytes[l] = pl.npad[l] / cg * 32;
            off += pl.wb_bytes[l];
        }
        off = round_up(off, 1024);
        if (pl.nslab[l] > maxslab) maxslab = pl.nslab[l];
        if (pl.npad[l] > maxn) maxn = pl.npad[l];
    }
    if (maxn > 256 || maxslab > MAX_SLABS) return false;            // two accumulators must fit the 512 TMEM columns
    pl.w_bytes_total = 0;
    for (int l = 0; l < n_linear; ++l) pl.w_bytes_total += (l == 0 ? 1 : pl.nslab[l]) * pl.w_slab_bytes[l] + pl.wb_bytes[l];
    pl.a0_off = off;
    off += 2 * A0_BYTES;
    pl.stage_off = off;
    off += IN_STAGES * STAGE_BYTES;
    pl.bias_base = off;
    off += round_up(pl.npad[n_linear - 1] * 4, 16);
    pl.bar_off = off;
    off += round_up(8 * B_COUNT + 8, 16);
    pl.red_off = off;
    off += 4 * HB_NMOM * 8;
    pl.total = off;
    pl.d_cols = round_up(maxn, 64);
    int cols = 32;
    while (cols < 2 * pl.d_cols) cols <<= 1;
    pl.tmem_cols = cols;
    return (size_t)pl.total + 1024 <= SMEM_LIMIT;
}

template <int CG, int ACT, bool F16, int G>
cudaError_t launch_one(const HbParticles& p, size_t n, const HbSurDev& sd, const TcPlan& pl, double* partials, int grid,
                       bool prepare, cudaStream_t s) {
    const size_t smem = (size_t)pl.total + 1024;   // slack so the 1024-byte alignment of the swizzle atoms always holds
    if (prepare)       // hb_lattice_finalize: the attribute is set once per lattice, not per push
        return cudaFuncSetAttribute(hb_sur_tc_kernel<CG, ACT, F16, G>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(tc_threads(G));
    cfg.dynamicSmemBytes = smem;
    cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = CG;
    at[0].val.clusterDim.y = 1;
    at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, hb_sur_tc_kernel<CG, ACT, F16, G>, p, n, sd, pl, partials);
}

template <int CG, bool F16, int G>
cudaError_t launch_act(const HbParticles& p, size_t n, const HbSurDev& sd, const TcPlan& pl, double* partials, int grid,
                       bool prepare, cudaStream_t s) {
    switch (sd.act) {
    case 0: return launch_one<CG, 0, F16, G>(p, n, sd, pl, partials, grid, prepare, s);
    case 1: return launch_one<CG, 1, F16, G>(p, n, sd, pl, partials, grid, prepare, s);
    case 2: return launch_one<CG, 2, F16, G>(p, n, sd, pl, partials, grid, prepare, s);
    default: return launch_one<CG, 3, F16, G>(p, n, sd, pl, partials, grid, prepare, s);
    }
}

template <int CG, bool F16>
cudaError_t launch_g(int g, const HbParticles& p, size_t n, const HbSurDev& sd, const TcPlan& pl, double* partials, int grid,
                     bool prepare, cudaStream_t s) {
    if (g == 1) return launch_act<CG, F16, 1>(p, n, sd, pl, partials, grid, prepare, s);
    return launch_act<CG, F16, 2>(p, n, sd, pl, partials, grid, prepare, s);
}

bool env_is(const char* name, char v) {
    const char* e = getenv(name);
    return e && e[0] == v;
}

}  // namespace

// Which kernel and launch shape a 16-bit / tf32 stage runs on.  Called ONCE per stage by hb_lattice_finalize (and by the
// host query hb_surrogate_kernel); the choice is stored in the segment, so nothing is decided per push.
//   kind 1  resident weights, one tile per CTA (this file): nets up to 128 wide run two CTAs per SM (G = 1: four
//           epilogue warps each; as single CTAs when the whole net fits one, else as pairs), the rest one CTA per SM
//   kind 4  resident weights, two tiles in flight per CTA (hb_sur_tc2.cu): hidden width above 128
//   kind 2  weights streamed from L2 (hb_sur_tcs.cu): nets that do not fit resident, and every HB_PREC_TF32 stage
//   kind 3  one launch per layer (hb_sur_tcw.cu): hidden widths 513..1024
// Test / tuning hooks read from the environment here and nowhere else: HB_TC_FORCE_CG=2 (CTA-pair shapes for nets that
// fit one CTA), HB_TC_FORCE_STREAM=1 (streamed kernel for nets that would stay resident), HB_TC_OCC2=0 (no
// two-CTAs-per-SM shape), HB_TC_ONE_TILE=1 (kind 1 where kind 4 would run).
HbTcChoice hb_tc_choose(int prec, int n_linear, const int* widths) {
    HbTcChoice ch{0, 0, 0, 0};
    if (prec < 1 || prec > 3) return ch;
    const bool force_cg2 = env_is("HB_TC_FORCE_CG", '2');
    TcPlan pl;
    int cg1 = 0;                                         // cluster size of the one-tile plan, 0 = does not fit
    if (prec != 3) {
        if (!force_cg2 && make_plan(1, n_linear, widths, pl)) cg1 = 1;
        else if (make_plan(2, n_linear, widths, pl)) cg1 = 2;
    }
    const int cg2 = prec == 3 ? 0 : hb_tc2_plan_cg(n_linear, widths, force_cg2 ? 2 : 0);
    const bool resident = cg1 != 0 || cg2 != 0;
    if (prec == 3 || (env_is("HB_TC_FORCE_STREAM", '1') && hb_tcs_supported(prec, n_linear, widths)) || !resident) {
        if (hb_tcs_supported(prec, n_linear, widths)) ch.kind = 2;
        else if (prec != 3 && hb_tcw_supported(prec, n_linear, widths)) ch.kind = 3;
        return ch;
    }
    if (cg2 != 0 && !(env_is("HB_TC_ONE_TILE", '1') && cg1 != 0)) {
        ch.kind = 4;
        ch.cg = cg2;
        ch.g = 2;
        ch.occ = 1;
        return ch;
    }
    ch.kind = 1;
    // two CTAs per SM for small plans: the second tile's MMAs fill the tensor pipe while the first is in its epilogue
    const bool allow_occ2 = !env_is("HB_TC_OCC2", '0') && !force_cg2;
    for (int cg = 1; cg <= 2 && allow_occ2; ++cg)
        if (make_plan(cg, n_linear, widths, pl) && (size_t)pl.total + 2048 <= SMEM_LIMIT / 2 && pl.tmem_cols <= 256) {
            ch.cg = cg; ch.g = 1; ch.occ = 2;
            return ch;
        }
    ch.cg = cg1; ch.g = 2; ch.occ = 1;
    return ch;
}

int hb_tc_kernel_kind(int prec, int n_linear, const int* widths) { return hb_tc_choose(prec, n_linear, widths).kind; }

bool hb_tc_supported(int prec, int n_linear, const int* widths, char* why, size_t why_len) {
    if (prec < 1 || prec > 3) {
        snprintf(why, why_len, "unknown precision %d", prec);
        return false;
    }
    if (hb_tc_choose(prec, n_linear, widths).kind != 0) return true;
    if (prec == 3)
        snprintf(why, why_len, "HB_PREC_TF32 runs on the streamed kernel only: at least one hidden layer, equal hidden widths <= 256");
    else
        snprintf(why, why_len, "no tensor-core schedule for this shape: the weights do not fit resident in shared memory "
                               "and the streamed / layered kernels need equal hidden widths <= 512 / <= 1024");
    return false;
}

// Packed operand image.  Layer 0 (K = 16, no swizzle): per 8-row group 256 bytes = K chunk 0 of the 8 rows
// (8 x 16 B) followed by K chunk 1; W_0 is carried twice (columns 0..5 multiply the hi parts of the inputs,
// 6..11 the lo parts).  Layers >= 1: per 64-wide K slab, npad rows of 128 bytes (K-major, 128-byte swizzle:
// the 16-byte chunk c of row r sits at chunk position c ^ (r mod 8)).
size_t hb_tc_pack_weights(const HbTcChoice& ch, int prec, int n_linear, const int* widths, const float* const* W,
                          const float* const* B, void* dst, long long* off_bytes, int* kpad, int* npad) {
    if (ch.kind == 2) return hb_tcs_pack_weights(prec, n_linear, widths, W, dst, off_bytes, kpad, npad);
    if (ch.kind == 3) return hb_tcw_pack_weights(prec, n_linear, widths, W, dst, off_bytes, kpad, npad);
    if (ch.kind == 4) return hb_tc2_pack_weights(prec, ch.cg, n_linear, widths, W, B, dst, off_bytes, kpad, npad);
    int ksteps[HB_MAX_LINEAR];
    layer_geometry(n_linear, widths, kpad, npad, ksteps);
    size_t total = 0;
    for (int l = 0; l < n_linear; ++l) {
        off_bytes[l] = (long long)total;
        total += l == 0 ? (size_t)npad[l] * 32 : (size_t)(kpad[l] / 64) * npad[l] * 128;
        if (l >= 1 && l + 1 < n_linear) total += (size_t)npad[l] * 32;      // bias block of a hidden layer
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
    // biases of layers 0 .. L-2 as b_hi, b_lo (value rounded to the operand type, rounded remainder) in K columns
    // 12, 13 of a K = 16 operand: inside W_0 for layer 0, in a block of its own behind the K slabs for the others
    for (int l = 0; l + 1 < n_linear; ++l) {
        const size_t blk = (size_t)off_bytes[l] + (l == 0 ? 0 : (size_t)(kpad[l] / 64) * npad[l] * 128);
        for (int o = 0; o < widths[l + 1]; ++o) {
            const unsigned short hi = bits16(B[l][o]);
            const unsigned short lo = bits16(B[l][o] - back32(hi));
            const size_t byte = blk + (size_t)(o / 8) * 256 + 128 + (size_t)(o % 8) * 16 + 4 * 2;   // k = 12
            std::memcpy(base + byte, &hi, 2);
            std::memcpy(base + byte + 2, &lo, 2);
        }
    }
    for (int l = 0; l < n_linear; ++l) {
        const int fin = widths[l], fout = widths[l + 1];
        const int kcols = l == 0 ? 12 : fin;
        for (int o = 0; o < fout; ++o)
            for (int k = 0; k < kcols; ++k) {
                const float w = l == 0 ? W[l][(size_t)o * fin + (k % 6)] : W[l][(size_t)o * fin + k];
                size_t byte;
                if (l == 0) {
                    byte = (size_t)off_bytes[l] + (size_t)(o / 8) * 256 + (size_t)(k / 8) * 128 + (size_t)(o % 8) * 16 + (size_t)(k % 8) * 2;
                } else {
                    const int slab = k / 64, kk = k % 64, c = kk / 8, e = kk % 8;
                    byte = (size_t)off_bytes[l] + (size_t)slab * npad[l] * 128 + (size_t)o * 128 +
                           (size_t)((c ^ (o & 7)) << 4) + (size_t)e * 2;
                }
                const unsigned short bits = bits16(w);
                std::memcpy(base + byte, &bits, 2);
            }
    }
    return total;
}

// prepare: only set the chosen kernel's shared-memory attribute (hb_lattice_finalize), launch nothing
cudaError_t hb_launch_sur_tc(const HbParticles& p, size_t n, const HbSurDev& sd, double* partials, int* nblocks_out,
                             int sm_count, bool prepare, cudaStream_t s) {
    if (sd.tc_kind == 2) return hb_launch_sur_tcs(p, n, sd, partials, nblocks_out, sm_count, prepare, s);
    if (sd.tc_kind == 4) return hb_launch_sur_tc2(p, n, sd, partials, nblocks_out, sm_count, prepare, s);
    TcPlan pl;
    const int cg = sd.tc_cg, g = sd.tc_g;
    if ((cg != 1 && cg != 2) || !make_plan(cg, sd.n_linear, sd.widths, pl)) return cudaErrorNotSupported;
    const size_t ntiles = (n + TILE_M - 1) / TILE_M;
    const size_t ngroups = (ntiles + cg - 1) / cg;
    size_t clusters = (size_t)(sm_count / cg) * sd.tc_occ;
    if (clusters > ngroups) clusters = ngroups;
    if (clusters < 1) clusters = 1;
    const int grid = (int)clusters * cg;
    if (nblocks_out) *nblocks_out = grid;
    const bool f16 = sd.prec == 2;
    if (cg == 1) return f16 ? launch_g<1, true>(g, p, n, sd, pl, partials, grid, prepare, s) : launch_g<1, false>(g, p, n, sd, pl, partials, grid, prepare, s);
    return f16 ? launch_g<2, true>(g, p, n, sd, pl, partials, grid, prepare, s) : launch_g<2, false>(g, p, n, sd, pl, partials, grid, prepare, s);
}
