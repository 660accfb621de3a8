// hb_sur_tcs.cu -- tensor-core surrogate stage (rows a4-a6) for networks whose weights do not fit in shared
// memory (hidden width up to 512, any depth: BJ config 5 is 6-512^4-6, 1.55 MB of 16-bit weights): the
// weights are STREAMED from L2 through a ring of 16 KB shared-memory blocks by the TMA engine while the
// activations of the tile stay on chip.
//
// A CTA pair (cta_group::2) owns 256 particles (128 TMEM lanes per CTA).  A hidden layer of padded width
// W = 2 * nh is computed as two N-halves h = 0, 1 with their own TMEM accumulators D_0, D_1 (2 x 256 columns =
// all of TMEM), K-slab by K-slab (64 inputs = one 16 KB weight block per CTA, four K = 16 MMAs):
//     (l,0,s0) .. (l,0,s7) | (l,1,s0) .. (l,1,s7)                       8192 tensor cycles at W = 512
// The epilogue of half 0 (tcgen05.ld, + bias, sigma, 16-bit, next A operand slabs 0..3) runs under the MMAs of
// half 1 -- slab j of the A buffer is overwritten once (l,1,s_j) has read it (A_FREE barriers) -- and the
// epilogue of half 1 (slabs 4..7) runs under (l+1,0,s0..s3), which only needs slabs 0..3.  The tensor pipe is
// never idle inside a tile as long as an epilogue half takes less time than four K slabs of MMAs.
// Warp roles (16 warps): 0-3 IO (prologue a4 / output a6 / moments a3), 4-11 hidden-layer epilogue,
// 12 particle-row producer (TMA), 13 weight producer (TMA ring), 14 relay (tells the leader CTA that this CTA's
// ring block has landed: a bulk copy cannot signal a barrier of the other CTA), 15 MMA issuer (leader CTA).
#include "hb_tc_common.cuh"

namespace {

constexpr int S_THREADS = 512;
constexpr int S_RING = 4;                        // weight ring slots
constexpr int S_BLOCK_BYTES = 16 * 1024;         // one slot: (nh / 2) rows x 128 B, nh <= 256
constexpr int S_MAX_SLABS = 8;                   // hidden width <= 512
enum : int {
    S_IN_FULL = 0,        // [2] coordinate rows staged (local)
    S_IN_EMPTY = 2,       // [2] stage consumed by the 4 IO warps (local)
    S_A0_FULL = 4,        // [2] layer-0 operand written (leader; 4 IO warps x 2 CTAs)
    S_RING_FULL = 6,      // [4] weight block landed (local, tx bytes)
    S_RING_EMPTY = 10,    // [4] weight block consumed (both CTAs, MMA commit)
    S_W_READY = 14,       // [4] weight block landed in both CTAs (leader; 2 relay arrivals)
    S_SLAB_FULL = 18,     // [8] K slab of the next A operand written (leader; 8 warps x 2 CTAs)
    S_A_FREE = 26,        // [4] slab j of the current A operand no longer read (both CTAs, MMA commit)
    S_D_FULL = 30,        // [2] accumulator half h of a hidden layer complete (both CTAs, MMA commit)
    S_D_LAST = 32,        // accumulator of the last layer complete (both CTAs, MMA commit)
    S_OUT_READ = 33,      // last layer's accumulator read by the IO warps (leader; 4 IO warps x 2 CTAs)
    S_COUNT = 34
};

struct TcsPlan {
    int n_linear;
    int npad;             // padded hidden width (all hidden layers), multiple of 128, <= 512
    int ns;               // npad / 64 : K slabs of a hidden operand
    int nh;               // npad / 2  : accumulator columns of one half
    int blk0_bytes;       // layer 0 block  : (npad / 2) rows x 32 B (this CTA's rows of both halves)
    int hblk_bytes;       // hidden block   : (nh / 2) rows x 128 B
    int last_bytes;       // last layer     : ns slabs x 8 rows x 128 B
    long long img_rank_bytes;   // bytes of one CTA rank's block sequence in the global image
    int bias_off[HB_MAX_LINEAR];
    int a_off, ring_off, a0_off, stage_off, bias_base, bar_off, red_off, total;
};

// EL: operand type  0 = bf16, 1 = f16 (kind::f16, 64 elements per 128-byte slab row, K = 16 per MMA),
//                   2 = tf32 (kind::tf32, 32 elements per slab row, K = 8 per MMA, half the rate; width <= 256)
template <int ACT, int EL>
__global__ void __launch_bounds__(S_THREADS, 1)
hb_sur_tcs_kernel(HbParticles p, size_t n, const __grid_constant__ HbSurDev sd, const __grid_constant__ TcsPlan pl,
                  double* __restrict__ partials) {
    constexpr int CG = 2;
    constexpr bool F16 = EL == 1, T32 = EL == 2;
    constexpr int A0B = T32 ? 2 * A0_BYTES : A0_BYTES;      // layer-0 operand buffer (K = 16 elements per row)
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    unsigned char* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    const uint32_t sbase = smem_u32(smem);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const uint32_t rank = cluster_rank();
    const size_t ntiles = (n + TILE_M - 1) / TILE_M;
    const size_t ngroups = (ntiles + CG - 1) / CG;
    const size_t cluster_id = blockIdx.x / CG, nclusters = gridDim.x / CG;
    const int L = pl.n_linear, NS = pl.ns, NS2 = pl.ns >> 1;

    const uint32_t bar0 = sbase + pl.bar_off;
    auto bar = [&](int i) -> uint32_t { return bar0 + 8u * (uint32_t)i; };
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + pl.bar_off + 8 * S_COUNT);
    float* bias_s = reinterpret_cast<float*>(smem + pl.bias_base);

    if (tid == 0) {
        for (int s = 0; s < 2; ++s) {
            mbar_init(bar(S_IN_FULL + s), 1);
            mbar_init(bar(S_IN_EMPTY + s), 4);
            mbar_init(bar(S_A0_FULL + s), 4 * CG);
            mbar_init(bar(S_D_FULL + s), 1);
        }
        for (int s = 0; s < S_RING; ++s) {
            mbar_init(bar(S_RING_FULL + s), 1);
            mbar_init(bar(S_RING_EMPTY + s), 1);
            mbar_init(bar(S_W_READY + s), CG);
            mbar_init(bar(S_A_FREE + s), 1);
        }
        for (int j = 0; j < S_MAX_SLABS; ++j) mbar_init(bar(S_SLAB_FULL + j), (T32 ? 4 : 8) * CG);
        mbar_init(bar(S_D_LAST), 1);
        mbar_init(bar(S_OUT_READ), 4 * CG);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 15) {
        tmem_alloc<CG>(smem_u32(tmem_slot), 512u);
        tmem_relinquish<CG>();
    }
    {   // biases -> shared (all layers)
        const int total = pl.bias_off[L - 1] + 16;
        for (int i = tid; i < total; i += S_THREADS) {
            int l = 0;
            while (l + 1 < L && i >= pl.bias_off[l + 1]) ++l;
            bias_s[i] = sd.btc[sd.btc_off[l] + (i - pl.bias_off[l])];
        }
    }
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;
    const int nblocks_tile = 2 + (L - 2) * 2 * NS;      // weight blocks one tile consumes

    if (warp == 12) {
        // ===================================================== particle-row producer
        if (lane == 0) {
            int stage = 0;
            uint32_t ph = 0;
            for (size_t g = cluster_id; g < ngroups; g += nclusters) {
                const size_t tile = g * CG + rank;
                const bool full = tile < ntiles && (tile + 1) * TILE_M <= n;
                if (full) {
                    mbar_wait<false>(bar(S_IN_EMPTY + stage), ph ^ 1);
                    mbar_expect_tx(bar(S_IN_FULL + stage), STAGE_BYTES);
                    for (int j = 0; j < 6; ++j)
                        bulk_g2s(sbase + pl.stage_off + stage * STAGE_BYTES + j * TILE_M * 4, p.v[j] + tile * TILE_M,
                                 TILE_M * 4, bar(S_IN_FULL + stage));
                    stage ^= 1;
                    if (stage == 0) ph ^= 1;
                }
            }
        }
        __syncwarp();
    } else if (warp == 13) {
        // ===================================================== weight producer: the block sequence of a tile,
        // over and over (layer 0 | (l, h, s) for l = 1..L-2 | last layer), through the ring
        if (lane == 0) {
            const unsigned char* img = reinterpret_cast<const unsigned char*>(sd.wtc) + (size_t)rank * (size_t)pl.img_rank_bytes;
            uint32_t cnt = 0;
            for (size_t g = cluster_id; g < ngroups; g += nclusters) {
                size_t off = 0;
                for (int b = 0; b < nblocks_tile; ++b, ++cnt) {
                    const uint32_t bytes = b == 0 ? (uint32_t)pl.blk0_bytes : (b == nblocks_tile - 1 ? (uint32_t)pl.last_bytes : (uint32_t)pl.hblk_bytes);
                    const uint32_t slot = cnt % S_RING, phs = (cnt / S_RING) & 1;
                    mbar_wait<false>(bar(S_RING_EMPTY + slot), phs ^ 1);
                    mbar_expect_tx(bar(S_RING_FULL + slot), bytes);
                    bulk_g2s(sbase + pl.ring_off + slot * S_BLOCK_BYTES, img + off, bytes, bar(S_RING_FULL + slot));
                    off += bytes;
                }
            }
        }
        __syncwarp();
    } else if (warp == 14) {
        // ===================================================== relay: block landed here -> tell the leader
        if (lane == 0) {
            uint32_t cnt = 0;
            for (size_t g = cluster_id; g < ngroups; g += nclusters)
                for (int b = 0; b < nblocks_tile; ++b, ++cnt) {
                    const uint32_t slot = cnt % S_RING, phs = (cnt / S_RING) & 1;
                    mbar_wait<true>(bar(S_RING_FULL + slot), phs);
                    mbar_arrive_cluster(bar(S_W_READY + slot), 0);
                }
        }
        __syncwarp();
    } else if (warp == 15) {
        // ===================================================== MMA issuer (leader CTA): warp-uniform walk of the
        // schedule, one elected lane issues
        if (rank == 0) {
            const uint32_t fmt = T32 ? 2u : (F16 ? 0u : 1u);
            const uint32_t idesc_base = (1u << 4) | (fmt << 7) | (fmt << 10) | ((uint32_t)((TILE_M * CG) >> 4) << 24);
            const uint32_t idesc_h = idesc_base | ((uint32_t)(pl.nh >> 3) << 17);
            const uint32_t idesc_last = idesc_base | ((uint32_t)(16 >> 3) << 17);
            const bool issuer = elect_one();
            const uint64_t a_desc0 = make_desc(sbase + pl.a_off);
            const uint32_t d0 = tmem_base, d1 = tmem_base + 256u;
            uint32_t cnt = 0;                        // weight blocks consumed so far
            uint32_t ph_slab = 0;                    // bit j: parity of the next completion of SLAB_FULL[j]
            uint32_t it = 0;
            auto wait_block = [&]() -> uint32_t {
                const uint32_t slot = cnt % S_RING;
                mbar_spin(bar(S_W_READY + slot), (cnt / S_RING) & 1);
                tc_fence_after();
                return slot;
            };
            auto release_block = [&](uint32_t slot) {
                if (issuer) umma_commit<CG>(bar(S_RING_EMPTY + slot));
                ++cnt;
            };
            auto wait_slab = [&](int j) {
                mbar_spin(bar(S_SLAB_FULL + j), (ph_slab >> j) & 1);
                ph_slab ^= 1u << j;
            };
            // slabs a layer needs before its MMA on slab s may go out.  s = 0: all of half 0's slabs -- the first
            // MMA overwrites D_0, which the epilogue of half 0 reads until it has written its last slab.
            auto wait_slabs_for = [&](int s) {
                if (s == 0) { for (int j = 0; j < NS2; ++j) wait_slab(j); }
                else if (s >= NS2) wait_slab(s);
                tc_fence_after();
            };
            for (size_t g = cluster_id; g < ngroups; g += nclusters, ++it) {
                // ---- layer 0: two N = nh MMAs (K = 16) from the compact operand buffers
                if (it > 0) mbar_spin(bar(S_OUT_READ), (it - 1) & 1);     // D_0[0..16) = previous outputs
                mbar_spin(bar(S_A0_FULL + (it & 1)), (it >> 1) & 1);
                {
                    const uint32_t slot = wait_block();
                    if (issuer) {
                        const uint32_t ab = sbase + pl.a0_off + (it & 1) * A0B;
                        const uint32_t wb = sbase + pl.ring_off + slot * S_BLOCK_BYTES;
                        if (T32) {      // K = 16 = two K = 8 MMAs; the second starts two core matrices (256 B) further
                            const uint64_t ad = make_desc_l0_t32(ab);
                            const uint64_t w0 = make_desc_l0_t32(wb), w1 = make_desc_l0_t32(wb + (uint32_t)(pl.nh >> 1) * 64u);
                            umma<CG, false, true>(d0, ad, w0, idesc_h);
                            umma<CG, true, true>(d0, ad + 16, w0 + 16, idesc_h);
                            umma_commit<CG>(bar(S_D_FULL + 0));
                            umma<CG, false, true>(d1, ad, w1, idesc_h);
                            umma<CG, true, true>(d1, ad + 16, w1 + 16, idesc_h);
                            umma_commit<CG>(bar(S_D_FULL + 1));
                        } else {
                            const uint64_t ad = make_desc_l0(ab);
                            umma<CG, false>(d0, ad, make_desc_l0(wb), idesc_h);
                            umma_commit<CG>(bar(S_D_FULL + 0));
                            umma<CG, false>(d1, ad, make_desc_l0(wb + (uint32_t)(pl.nh >> 1) * 32u), idesc_h);
                            umma_commit<CG>(bar(S_D_FULL + 1));
                        }
                    }
                    release_block(slot);
                    __syncwarp();
                }
                // ---- hidden layers 1 .. L-2
                for (int l = 1; l < L - 1; ++l) {
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        const uint32_t d_tmem = h ? d1 : d0;
#pragma unroll
                        for (int s = 0; s < S_MAX_SLABS; ++s) {
                            if (s < NS) {
                                if (h == 0) wait_slabs_for(s);
                                const uint32_t slot = wait_block();
                                if (issuer) {
                                    const uint64_t ad = a_desc0 + (uint64_t)(s * (A_SLAB_BYTES >> 4));
                                    const uint64_t bd = make_desc(sbase + pl.ring_off + slot * S_BLOCK_BYTES);
                                    if (s == 0) umma<CG, false, T32>(d_tmem, ad, bd, idesc_h);
                                    else umma<CG, true, T32>(d_tmem, ad, bd, idesc_h);
                                    umma<CG, true, T32>(d_tmem, ad + 2, bd + 2, idesc_h);
                                    umma<CG, true, T32>(d_tmem, ad + 4, bd + 4, idesc_h);
                                    umma<CG, true, T32>(d_tmem, ad + 6, bd + 6, idesc_h);
                                }
                                release_block(slot);
                                // half 1 has read slab s: the epilogue of half 0 may overwrite it
                                if (h == 1 && s < NS2 && issuer) umma_commit<CG>(bar(S_A_FREE + s));
                                __syncwarp();
                            }
                        }
                        if (issuer) umma_commit<CG>(bar(S_D_FULL + h));
                        __syncwarp();
                    }
                }
                // ---- last layer: N = 16 into D_0[0..16), all K slabs from one ring block
                {
                    const uint32_t slot = wait_block();
#pragma unroll
                    for (int s = 0; s < S_MAX_SLABS; ++s) {
                        if (s < NS) {
                            wait_slabs_for(s);
                            if (issuer) {
                                const uint64_t ad = a_desc0 + (uint64_t)(s * (A_SLAB_BYTES >> 4));
                                const uint64_t bd = make_desc(sbase + pl.ring_off + slot * S_BLOCK_BYTES + s * 1024);
                                if (s == 0) umma<CG, false, T32>(d0, ad, bd, idesc_last);
                                else umma<CG, true, T32>(d0, ad, bd, idesc_last);
                                umma<CG, true, T32>(d0, ad + 2, bd + 2, idesc_last);
                                umma<CG, true, T32>(d0, ad + 4, bd + 4, idesc_last);
                                umma<CG, true, T32>(d0, ad + 6, bd + 6, idesc_last);
                            }
                            __syncwarp();
                        }
                    }
                    if (issuer) umma_commit<CG>(bar(S_D_LAST));
                    release_block(slot);
                    __syncwarp();
                }
            }
        }
        __syncwarp();
    } else if (warp < 4) {
        // ===================================================== IO warps: prologue of tile i+1, output of tile i
        const int row = 32 * warp + lane;        // tile row = TMEM lane = particle within the tile
        const uint32_t a0_row = sbase + pl.a0_off + (uint32_t)(row >> 3) * 256 + (uint32_t)(row & 7) * 16;
        const uint32_t tlane = tmem_base + ((uint32_t)(32 * warp) << 16);
        const float* bl = bias_s + pl.bias_off[L - 1];
        HbMomAcc acc;
        acc.clear();
        int stage = 0;
        uint32_t pin = 0;
        auto prologue = [&](size_t g, uint32_t buf) {
            const size_t tile = g * CG + rank;
            const size_t i = tile * TILE_M + row;
            const bool valid = tile < ntiles && i < n;
            const bool full = tile < ntiles && (tile + 1) * TILE_M <= n;
            float c[6] = {0, 0, 0, 0, 0, 0};
            if (full) {
                mbar_wait<false>(bar(S_IN_FULL + stage), pin);
                const float* st = reinterpret_cast<const float*>(smem + pl.stage_off + stage * STAGE_BYTES);
#pragma unroll
                for (int j = 0; j < 6; ++j) c[j] = st[j * TILE_M + row];
                __syncwarp();
                if (lane == 0) mbar_arrive_local(bar(S_IN_EMPTY + stage));
                stage ^= 1;
                if (stage == 0) pin ^= 1;
            } else if (valid) {
#pragma unroll
                for (int j = 0; j < 6; ++j) c[j] = p.v[j][i];
            }
            if (T32) {   // 8-row groups of 512 B: four K chunks (4 elements each) 128 B apart
                uint32_t q[4][4];
                tc_make_a0_row_t32(sd, valid, c, q);
                const uint32_t dst = sbase + pl.a0_off + buf * A0B + (uint32_t)(row >> 3) * 512 + (uint32_t)(row & 7) * 16;
#pragma unroll
                for (int k = 0; k < 4; ++k) sts128(dst + 128 * k, q[k]);
            } else {
                uint32_t q0[4], q1[4];
                tc_make_a0_row<F16>(sd, valid, c, q0, q1);
                const uint32_t dst = a0_row + buf * A0B;
                sts128(dst, q0);
                sts128(dst + 128, q1);
            }
            fence_proxy_async();
            __syncwarp();
            if (lane == 0) mbar_arrive_cluster(bar(S_A0_FULL + buf), 0);
        };
        uint32_t it = 0;
        if (cluster_id < ngroups) prologue(cluster_id, 0);
        for (size_t g = cluster_id; g < ngroups; g += nclusters, ++it) {
            if (g + nclusters < ngroups) prologue(g + nclusters, (it + 1) & 1);
            const size_t tile = g * CG + rank;
            const size_t i = tile * TILE_M + row;
            const bool valid = tile < ntiles && i < n;
            mbar_wait<false>(bar(S_D_LAST), it & 1);
            tc_fence_after();
            uint32_t r[8];
            tmem_ld8(tlane, r);
            tmem_ld_wait();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive_cluster(bar(S_OUT_READ), 0);
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
            hb_block_reduce_moments(acc, red, partials + blockIdx.x, tid, 128, 2);
        }
    } else if (warp < 12) {
        // ===================================================== hidden-layer epilogue warps
        const int wq = warp & 3;
        const int grp = (warp - 4) >> 2;          // 32-column group inside every 64-column slab
        const int row = 32 * wq + lane;
        const uint32_t a_row = sbase + pl.a_off + row * 128;
        const uint32_t sw = (uint32_t)(row & 7);
        const uint32_t tlane = tmem_base + ((uint32_t)(32 * wq) << 16);
        uint32_t ph_d = 0;                        // bit h: parity of the next completion of D_FULL[h]
        uint32_t ph_free = 0;                     // bit j: parity of the next completion of A_FREE[j]
        for (size_t g = cluster_id; g < ngroups; g += nclusters) {
            for (int l = 0; l < L - 1; ++l) {
                const float* bl = bias_s + pl.bias_off[l];
                const float slope = sd.prelu[l];
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    mbar_wait<true>(bar(S_D_FULL + h), (ph_d >> h) & 1);
                    ph_d ^= 1u << h;
                    tc_fence_after();
                    // this warp's 32-column chunks of the half: c = grp, grp + 2, ...  (16-bit operands: chunk c is
                    // half of slab c / 2; tf32: chunk c is slab c)
                    const int nchunk = pl.nh >> 5;
                    auto finish = [&](const uint32_t (&r)[32], int c) {
                        const int slab_in_half = T32 ? c : (c >> 1);
                        const int slab = h * NS2 + slab_in_half;
                        if (h == 0 && l > 0) {        // half 1's MMAs must have read this slab of the current operand
                            if (T32 || grp == (c & 1)) {   // (every chunk of this warp lies in a different slab)
                                mbar_wait<true>(bar(S_A_FREE + slab_in_half), (ph_free >> slab_in_half) & 1);
                                ph_free ^= 1u << slab_in_half;
                            }
                        }
                        if (T32) epi_store_t32<ACT>(r, bl + h * pl.nh + 32 * c, slope, a_row + slab * A_SLAB_BYTES, sw);
                        else epi_store<32, ACT, F16>(r, bl, h * pl.nh + 32 * c, slope, a_row, sw);
                        fence_proxy_async();
                        tc_fence_before();
                        __syncwarp();
                        if (lane == 0) mbar_arrive_cluster(bar(S_SLAB_FULL + slab), 0);
                    };
                    uint32_t ra[32], rb[32];
                    const uint32_t tb = tlane + (uint32_t)(h * 256);
                    tmem_ld32(tb + 32 * grp, ra);
                    for (int c = grp; c < nchunk; c += 4) {
                        tmem_ld_wait();
                        if (c + 2 < nchunk) tmem_ld32(tb + 32 * (c + 2), rb);
                        finish(ra, c);
                        if (c + 2 < nchunk) {
                            tmem_ld_wait();
                            if (c + 4 < nchunk) tmem_ld32(tb + 32 * (c + 4), ra);
                            finish(rb, c + 2);
                        }
                    }
                }
            }
        }
    }
    // ---- teardown: everyone done with TMEM (both CTAs of the pair), then free it
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();
    if (warp == 15) {
        tc_fence_after();
        tmem_dealloc<CG>(tmem_base, 512u);
    }
}

// ------------------------------------------------------------------------------- host: plan + packing
int s_round_up(int v, int m) { return (v + m - 1) / m * m; }

bool make_splan(int prec, int n_linear, const int* widths, TcsPlan& pl) {
    const bool t32 = prec == 3;
    std::memset(&pl, 0, sizeof pl);
    if (n_linear < 2) return false;
    int npad = 0;
    for (int l = 0; l < n_linear - 1; ++l) {
        const int w = s_round_up(widths[l + 1], 128);
        if (l == 0) npad = w;
        else if (w != npad) return false;                            // equal (padded) hidden widths only
    }
    if (npad > (t32 ? 256 : 512)) return false;      // operand buffer: 8 slabs of 64 (16-bit) or 32 (tf32) inputs
    pl.n_linear = n_linear;
    pl.npad = npad;
    pl.ns = npad / (t32 ? 32 : 64);
    pl.nh = npad / 2;
    pl.blk0_bytes = npad / 2 * (t32 ? 64 : 32);
    pl.hblk_bytes = pl.nh / 2 * 128;
    pl.last_bytes = pl.ns * 1024;
    pl.img_rank_bytes = (long long)pl.blk0_bytes + (long long)(n_linear - 2) * 2 * pl.ns * pl.hblk_bytes + pl.last_bytes;
    int boff = 0;
    for (int l = 0; l < n_linear; ++l) {
        pl.bias_off[l] = boff;
        boff += l == n_linear - 1 ? 16 : npad;
    }
    int off = 0;
    pl.a_off = off;
    off += pl.ns * A_SLAB_BYTES;
    pl.ring_off = off;
    off += S_RING * S_BLOCK_BYTES;
    pl.a0_off = off;
    off += 2 * (t32 ? 2 * A0_BYTES : A0_BYTES);
    pl.stage_off = off;
    off += IN_STAGES * STAGE_BYTES;
    pl.bias_base = off;
    off += s_round_up(boff * 4, 16);
    pl.bar_off = off;
    off += s_round_up(8 * S_COUNT + 8, 16);
    pl.red_off = off;
    off += 4 * HB_NMOM * 8;
    pl.total = off;
    return (size_t)pl.total + 1024 <= SMEM_LIMIT;
}

template <int ACT, int EL>
cudaError_t s_launch_one(const HbParticles& p, size_t n, const HbSurDev& sd, const TcsPlan& pl, double* partials, int grid,
                         bool prepare, cudaStream_t s) {
    const size_t smem = (size_t)pl.total + 1024;
    if (prepare) return cudaFuncSetAttribute(hb_sur_tcs_kernel<ACT, EL>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(S_THREADS);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = 2;
    at[0].val.clusterDim.y = 1;
    at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, hb_sur_tcs_kernel<ACT, EL>, p, n, sd, pl, partials);
}

template <int EL>
cudaError_t s_launch_act(const HbParticles& p, size_t n, const HbSurDev& sd, const TcsPlan& pl, double* partials, int grid,
                         bool prepare, cudaStream_t s) {
    switch (sd.act) {
    case 0: return s_launch_one<0, EL>(p, n, sd, pl, partials, grid, prepare, s);
    case 1: return s_launch_one<1, EL>(p, n, sd, pl, partials, grid, prepare, s);
    case 2: return s_launch_one<2, EL>(p, n, sd, pl, partials, grid, prepare, s);
    default: return s_launch_one<3, EL>(p, n, sd, pl, partials, grid, prepare, s);
    }
}

}  // namespace

bool hb_tcs_supported(int prec, int n_linear, const int* widths) {
    TcsPlan pl;
    return make_splan(prec, n_linear, widths, pl);
}

// Global image = [rank 0 block sequence | rank 1 block sequence]; a rank's sequence is what its weight producer
// walks per tile: layer 0 block, hidden blocks (l, h, s), last-layer block.  CTA `rank` holds, of half h, the rows
// of neurons h*nh + rank*nh/2 + i (i < nh/2), i.e. accumulator column rank*nh/2 + i of D_h.
//   layer 0 block : rows [half 0 | half 1], K = 16 no-swizzle (8-row groups of 256 B: K chunk 0, K chunk 1)
//   hidden block  : nh/2 rows x 128 B, K-major 128-byte swizzle (chunk c of row r at c ^ (r mod 8))
//   last block    : per K slab 8 rows x 128 B (rank 0: outputs 0..7, rank 1: outputs 8..15), swizzled
size_t hb_tcs_pack_weights(int prec, int n_linear, const int* widths, const float* const* W, void* dst,
                           long long* off_bytes, int* kpad, int* npad) {
    TcsPlan pl;
    if (!make_splan(prec, n_linear, widths, pl)) return 0;
    const bool t32 = prec == 3;
    const int ks = t32 ? 32 : 64;                    // inputs per slab
    const int esz = t32 ? 4 : 2;
    for (int l = 0; l < n_linear; ++l) {
        off_bytes[l] = 0;                                    // the kernel walks the block sequence itself
        npad[l] = l == n_linear - 1 ? 16 : pl.npad;
        kpad[l] = l == 0 ? 16 : pl.npad;
    }
    const size_t total = 2 * (size_t)pl.img_rank_bytes;
    if (!dst) return total;
    std::memset(dst, 0, total);
    unsigned char* base = static_cast<unsigned char*>(dst);
    // element e of a 16-byte chunk starting at `chunk_byte`
    auto put = [&](size_t chunk_byte, int e, float w) {
        if (t32) {           // tf32: fp32 container, 10 explicit mantissa bits, round to nearest (ties away)
            unsigned int u;
            std::memcpy(&u, &w, 4);
            u = (u + 0x1000u) & 0xffffe000u;
            std::memcpy(base + chunk_byte + (size_t)e * 4, &u, 4);
            return;
        }
        unsigned short bits;
        if (prec == 2) { __half h = __float2half_rn(w); std::memcpy(&bits, &h, 2); }
        else { __nv_bfloat16 h = __float2bfloat16_rn(w); std::memcpy(&bits, &h, 2); }
        std::memcpy(base + chunk_byte + (size_t)e * 2, &bits, 2);
    };
    const int epc = 16 / esz;                        // elements per 16-byte chunk
    const int nh = pl.nh, nq = pl.nh / 2;
    for (int rank = 0; rank < 2; ++rank) {
        const size_t r0 = (size_t)rank * (size_t)pl.img_rank_bytes;
        // layer 0
        for (int h = 0; h < 2; ++h)
            for (int i = 0; i < nq; ++i) {
                const int o = h * nh + rank * nq + i;
                if (o >= widths[1]) continue;
                const int row = h * nq + i;
                // K = 16 no-swizzle: per 8-row group, K chunk c (epc elements) at c * 128 B
                for (int k = 0; k < 12; ++k)
                    put(r0 + (size_t)(row / 8) * (size_t)(16 / epc * 128) + (size_t)(k / epc) * 128 + (size_t)(row % 8) * 16, k % epc,
                        W[0][(size_t)o * widths[0] + (k % 6)]);
            }
        // hidden layers
        for (int l = 1; l < n_linear - 1; ++l)
            for (int h = 0; h < 2; ++h)
                for (int s = 0; s < pl.ns; ++s) {
                    const size_t b0 = r0 + (size_t)pl.blk0_bytes + ((size_t)((l - 1) * 2 + h) * pl.ns + s) * (size_t)pl.hblk_bytes;
                    for (int i = 0; i < nq; ++i) {
                        const int o = h * nh + rank * nq + i;
                        if (o >= widths[l + 1]) continue;
                        for (int kk = 0; kk < ks; ++kk) {
                            const int k = s * ks + kk;
                            if (k >= widths[l]) break;
                            put(b0 + (size_t)i * 128 + (size_t)(((kk / epc) ^ (i & 7)) << 4), kk % epc,
                                W[l][(size_t)o * widths[l] + k]);
                        }
                    }
                }
        // last layer
        {
            const int l = n_linear - 1;
            const size_t b0 = r0 + (size_t)pl.blk0_bytes + (size_t)(n_linear - 2) * 2 * pl.ns * (size_t)pl.hblk_bytes;
            for (int i = 0; i < 8; ++i) {
                const int o = rank * 8 + i;
                if (o >= widths[l + 1]) continue;
                for (int k = 0; k < widths[l]; ++k) {
                    const int s = k / ks, kk = k % ks;
                    put(b0 + (size_t)s * 1024 + (size_t)i * 128 + (size_t)(((kk / epc) ^ (i & 7)) << 4), kk % epc,
                        W[l][(size_t)o * widths[l] + k]);
                }
            }
        }
    }
    return total;
}

cudaError_t hb_launch_sur_tcs(const HbParticles& p, size_t n, const HbSurDev& sd, double* partials, int* nblocks_out,
                              int sm_count, bool prepare, cudaStream_t s) {
    TcsPlan pl;
    if (!make_splan(sd.prec, sd.n_linear, sd.widths, pl)) return cudaErrorNotSupported;
    const size_t ntiles = (n + TILE_M - 1) / TILE_M;
    const size_t ngroups = (ntiles + 1) / 2;
    size_t clusters = (size_t)(sm_count / 2);
    if (clusters > ngroups) clusters = ngroups;
    if (clusters < 1) clusters = 1;
    const int grid = (int)clusters * 2;
    if (nblocks_out) *nblocks_out = grid;
    if (sd.prec == 3) return s_launch_act<2>(p, n, sd, pl, partials, grid, prepare, s);
    return sd.prec == 2 ? s_launch_act<1>(p, n, sd, pl, partials, grid, prepare, s) : s_launch_act<0>(p, n, sd, pl, partials, grid, prepare, s);
}
