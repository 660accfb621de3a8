// hb_sur_tcw.cu -- tensor-core surrogate stage (rows a4-a6) for WIDE networks (hidden width 513..1024, equal
// widths: the paper's own 6-900^5-6 and 6-700^3-6 nets), one kernel launch per linear layer.
//
// A 128-particle tile of a 1024-wide layer needs 256 KB of 16-bit operand and 1024 accumulator columns: neither
// shared memory (227 KB) nor TMEM (512 columns) holds a whole layer, so the activations of a chunk of particles
// round-trip through two global scratch buffers (L2 / HBM) between layer kernels.  The scratch is stored PRE-TILED:
// per CTA (128 particles of a 256-particle pair tile) and 64-feature K slab one contiguous 16 KB block that already
// is the 128-byte-swizzled K-major operand image, so a slab moves with one cp.async.bulk each way.
// Per layer, per pair tile, per 256-column output block nb:  for every K slab s a ring stage receives
// (A slab of the tile, W block (nb, s)) = 32 KB, four K = 16 MMAs accumulate into D[nb & 1]; the epilogue of block
// nb (tcgen05.ld, + bias, sigma, 16 bit, staging slab, bulk store to the output scratch) runs under the MMAs of
// block nb+1.  The first layer takes its K = 16 operand from the fused prologue (a4), the last layer (N = 16) feeds
// the fused output epilogue (a6) and the moments (a3), as in hb_sur_tcs.cu.
// Warp roles (16 warps): 0-3 IO, 4-11 epilogue, 12 idle, 13 producer (TMA ring), 14 relay, 15 MMA issuer.
#include "hb_tc_common.cuh"

#include <algorithm>

namespace {

constexpr int W_THREADS = 512;
constexpr int W_RING = 5;                        // ring stages of 32 KB: A slab (16 KB) + W block (16 KB)
constexpr int W_STAGE_BYTES = 32 * 1024;
enum : int {
    Q_A0_FULL = 0,        // [2] layer-0 operand written (leader; 4 IO warps x 2 CTAs)            (first layer)
    Q_RING_FULL = 2,      // [5] stage landed (local, tx bytes)
    Q_RING_EMPTY = 7,     // [5] stage consumed (both CTAs, MMA commit)
    Q_W_READY = 12,       // [5] stage landed in both CTAs (leader; 2 relay arrivals)
    Q_D_FULL = 17,        // [2] accumulator D[b] complete (both CTAs, MMA commit)
    Q_D_FREE = 19,        // [2] accumulator D[b] read by the epilogue (leader; 8 warps x 2 CTAs)
    Q_D_LAST = 21,        // last layer: outputs complete (both CTAs, MMA commit)
    Q_OUT_READ = 22,      // last layer: outputs read by the IO warps (leader; 4 x 2)
    Q_A0_FREE = 23,       // [2] first layer: the MMAs of a tile have read its layer-0 operand buffer (both, commit)
    Q_COUNT = 25
};

struct TcwPlan {
    int npad;             // padded hidden width, multiple of 64, <= 1024
    int ns;               // npad / 64  K slabs of a hidden operand
    int nb;               // ceil(npad / 256) output blocks of a hidden layer: 256 columns each, the last one the rest
    int ring_off, stage_out_off, a0_off, bias_off, bar_off, red_off, total;
};

// what one launch does
struct TcwLayer {
    int first, last;              // first: operand from the particles (K = 16); last: N = 16, outputs to the particles
    int layer;                    // index l of the linear map (bias, PReLU slope)
    long long w_off;              // byte offset of this layer's block sequence of rank 0 in the weight image
    long long w_rank_bytes;       // bytes of one rank's block sequence of this layer
    const unsigned char* act_in;  // pre-tiled activations of the chunk (unused if first)
    unsigned char* act_out;       // (unused if last)
    size_t row_off;               // first particle of the chunk in the bunch (particle arrays are NOT offset)
};

__device__ __forceinline__ void bulk_s2g(void* dst, uint32_t src, uint32_t bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(src), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }

template <int ACT, bool F16>
__global__ void __launch_bounds__(W_THREADS, 1)
hb_sur_tcw_kernel(HbParticles p, size_t n_chunk, const __grid_constant__ HbSurDev sd, const __grid_constant__ TcwPlan pl,
                  const __grid_constant__ TcwLayer ly, double* __restrict__ partials) {
    constexpr int CG = 2;
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    unsigned char* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    const uint32_t sbase = smem_u32(smem);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const uint32_t rank = cluster_rank();
    const size_t ntiles = (n_chunk + TILE_M - 1) / TILE_M;       // tiles of this chunk
    const size_t ngroups = (ntiles + CG - 1) / CG;
    const size_t cluster_id = blockIdx.x / CG, nclusters = gridDim.x / CG;
    const int NS = pl.ns;
    const int NB = ly.last ? 1 : pl.nb;              // output blocks of this layer
    const int KS = ly.first ? 1 : NS;                // ring stages per output block

    const uint32_t bar0 = sbase + pl.bar_off;
    auto bar = [&](int i) -> uint32_t { return bar0 + 8u * (uint32_t)i; };
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + pl.bar_off + 8 * Q_COUNT);
    float* bias_s = reinterpret_cast<float*>(smem + pl.bias_off);

    if (tid == 0) {
        for (int s = 0; s < 2; ++s) {
            mbar_init(bar(Q_A0_FULL + s), 4 * CG);
            mbar_init(bar(Q_A0_FREE + s), 1);
            mbar_init(bar(Q_D_FULL + s), 1);
            mbar_init(bar(Q_D_FREE + s), 8 * CG);
        }
        for (int s = 0; s < W_RING; ++s) {
            mbar_init(bar(Q_RING_FULL + s), 1);
            mbar_init(bar(Q_RING_EMPTY + s), 1);
            mbar_init(bar(Q_W_READY + s), CG);
        }
        mbar_init(bar(Q_D_LAST), 1);
        mbar_init(bar(Q_OUT_READ), 4 * CG);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 15) {
        tmem_alloc<CG>(smem_u32(tmem_slot), 512u);
        tmem_relinquish<CG>();
    }
    {   // biases of this layer -> shared
        const int total = ly.last ? 16 : pl.npad;
        for (int i = tid; i < total; i += W_THREADS) bias_s[i] = sd.btc[sd.btc_off[ly.layer] + i];
    }
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    // output block nb is 256 columns wide, the last one what is left of npad; this CTA holds half of its weight rows
    auto blk_w = [&](int nb) -> int { return ly.last ? 16 : min(256, pl.npad - 256 * nb); };
    // bytes of the weight part of a stage of block nb (full blocks precede the narrow one, so nb * full size = offset)
    auto w_bytes_of = [&](int nb) -> uint32_t {
        return ly.last ? 1024u : (uint32_t)(blk_w(nb) / 2) * (ly.first ? 32u : 128u);
    };
    const uint32_t w_full = ly.first ? 128u * 32u : (ly.last ? 1024u : 16384u);
    const unsigned char* wimg = reinterpret_cast<const unsigned char*>(sd.wtc) + ly.w_off + (size_t)rank * (size_t)ly.w_rank_bytes;

    if (warp == 13) {
        // ===================================================== producer: (A slab, W block) per stage, order (tile, nb, s)
        if (lane == 0) {
            uint32_t cnt = 0;
            for (size_t g = cluster_id; g < ngroups; g += nclusters) {
                const unsigned char* a_tile = ly.first ? nullptr : ly.act_in + ((g * CG + rank) * (size_t)NS) * A_SLAB_BYTES;
                for (int nb = 0; nb < NB; ++nb) {
                    const uint32_t w_bytes = w_bytes_of(nb);
                    for (int s = 0; s < KS; ++s, ++cnt) {
                        const uint32_t slot = cnt % W_RING, phs = (cnt / W_RING) & 1;
                        mbar_wait<false>(bar(Q_RING_EMPTY + slot), phs ^ 1);
                        const uint32_t dst = sbase + pl.ring_off + slot * W_STAGE_BYTES;
                        mbar_expect_tx(bar(Q_RING_FULL + slot), (ly.first ? 0u : (uint32_t)A_SLAB_BYTES) + w_bytes);
                        if (!ly.first) bulk_g2s(dst, a_tile + (size_t)s * A_SLAB_BYTES, A_SLAB_BYTES, bar(Q_RING_FULL + slot));
                        bulk_g2s(dst + A_SLAB_BYTES, wimg + (size_t)nb * KS * w_full + (size_t)s * w_bytes, w_bytes, bar(Q_RING_FULL + slot));
                    }
                }
            }
        }
        __syncwarp();
    } else if (warp == 14) {
        // ===================================================== relay: stage landed here -> tell the leader
        if (lane == 0) {
            uint32_t cnt = 0;
            for (size_t g = cluster_id; g < ngroups; g += nclusters)
                for (int b = 0; b < NB * KS; ++b, ++cnt) {
                    const uint32_t slot = cnt % W_RING, phs = (cnt / W_RING) & 1;
                    mbar_wait<true>(bar(Q_RING_FULL + slot), phs);
                    mbar_arrive_cluster(bar(Q_W_READY + slot), 0);
                }
        }
        __syncwarp();
    } else if (warp == 15) {
        // ===================================================== MMA issuer (leader CTA)
        if (rank == 0) {
            const uint32_t fmt = F16 ? 0u : 1u;
            const uint32_t idesc_base = (1u << 4) | (fmt << 7) | (fmt << 10) | ((uint32_t)((TILE_M * CG) >> 4) << 24);
            const bool issuer = elect_one();
            uint32_t cnt = 0;                        // ring stages consumed
            uint32_t use[2] = {0, 0};                // how often D[b] has been filled so far
            uint32_t it = 0;
            for (size_t g = cluster_id; g < ngroups; g += nclusters, ++it) {
                if (ly.first) mbar_spin(bar(Q_A0_FULL + (it & 1)), (it >> 1) & 1);
                if (ly.last && it > 0) mbar_spin(bar(Q_OUT_READ), (it - 1) & 1);   // D[0][0..16) = previous outputs
                for (int nb = 0; nb < NB; ++nb) {
                    const uint32_t b = (uint32_t)nb & 1u;
                    const uint32_t d_tmem = tmem_base + b * 256u;
                    const uint32_t idesc = idesc_base | ((uint32_t)(blk_w(nb) >> 3) << 17);
                    // the epilogue must have read the block that filled D[b] before
                    if (!ly.last && use[b] > 0) mbar_spin(bar(Q_D_FREE + b), (use[b] - 1) & 1);
                    ++use[b];
                    for (int s = 0; s < KS; ++s, ++cnt) {
                        const uint32_t slot = cnt % W_RING;
                        mbar_spin(bar(Q_W_READY + slot), (cnt / W_RING) & 1);
                        tc_fence_after();
                        if (issuer) {
                            const uint32_t st = sbase + pl.ring_off + slot * W_STAGE_BYTES;
                            if (ly.first) {
                                umma<CG, false>(d_tmem, make_desc_l0(sbase + pl.a0_off + (it & 1) * A0_BYTES),
                                                make_desc_l0(st + A_SLAB_BYTES), idesc);
                            } else {
                                const uint64_t ad = make_desc(st), bd = make_desc(st + A_SLAB_BYTES);
                                if (s == 0) umma<CG, false>(d_tmem, ad, bd, idesc);
                                else umma<CG, true>(d_tmem, ad, bd, idesc);
                                umma<CG, true>(d_tmem, ad + 2, bd + 2, idesc);
                                umma<CG, true>(d_tmem, ad + 4, bd + 4, idesc);
                                umma<CG, true>(d_tmem, ad + 6, bd + 6, idesc);
                            }
                            umma_commit<CG>(bar(Q_RING_EMPTY + slot));
                        }
                        __syncwarp();
                    }
                    if (issuer) umma_commit<CG>(ly.last ? bar(Q_D_LAST) : bar(Q_D_FULL + b));
                    __syncwarp();
                }
                if (ly.first && issuer) umma_commit<CG>(bar(Q_A0_FREE + (it & 1)));
                __syncwarp();
            }
        }
        __syncwarp();
    } else if (warp < 4) {
        // ===================================================== IO warps: prologue (first layer) / output (last layer)
        const int row = 32 * warp + lane;
        const uint32_t a0_row = sbase + pl.a0_off + (uint32_t)(row >> 3) * 256 + (uint32_t)(row & 7) * 16;
        const uint32_t tlane = tmem_base + ((uint32_t)(32 * warp) << 16);
        HbMomAcc acc;
        acc.clear();
        if (ly.first) {
            uint32_t it = 0;
            for (size_t g = cluster_id; g < ngroups; g += nclusters, ++it) {
                const size_t tile = g * CG + rank;
                const size_t i = tile * TILE_M + row;
                const bool valid = i < n_chunk;
                float c[6] = {0, 0, 0, 0, 0, 0};
                if (valid) {
#pragma unroll
                    for (int j = 0; j < 6; ++j) c[j] = __ldcs(p.v[j] + ly.row_off + i);
                }
                uint32_t q0[4], q1[4];
                tc_make_a0_row<F16>(sd, valid, c, q0, q1);
                // buffer (it & 1) was last read by the layer-0 MMAs of tile it-2
                if (it >= 2) mbar_wait<false>(bar(Q_A0_FREE + (it & 1)), ((it >> 1) - 1) & 1);
                const uint32_t dst = a0_row + (it & 1) * A0_BYTES;
                sts128(dst, q0);
                sts128(dst + 128, q1);
                fence_proxy_async();
                __syncwarp();
                if (lane == 0) mbar_arrive_cluster(bar(Q_A0_FULL + (it & 1)), 0);
            }
        }
        if (ly.last) {
            float bl[6];
#pragma unroll
            for (int j = 0; j < 6; ++j) bl[j] = bias_s[j];
            uint32_t it = 0;
            for (size_t g = cluster_id; g < ngroups; g += nclusters, ++it) {
                const size_t tile = g * CG + rank;
                const size_t i = tile * TILE_M + row;
                const bool valid = i < n_chunk;
                mbar_wait<false>(bar(Q_D_LAST), it & 1);
                tc_fence_after();
                uint32_t r[8];
                tmem_ld8(tlane, r);
                tmem_ld_wait();
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive_cluster(bar(Q_OUT_READ), 0);
                if (valid) {
                    float w[6];
#pragma unroll
                    for (int j = 0; j < 6; ++j) w[j] = __uint_as_float(r[j]) + bl[j];
                    float x, px, y, py, t, pt;
                    hb_sur_epilogue(sd, w, x, px, y, py, t, pt);
                    const size_t o = ly.row_off + i;
                    p.v[0][o] = x; p.v[1][o] = px; p.v[2][o] = y; p.v[3][o] = py; p.v[4][o] = t; p.v[5][o] = pt;
                    if (partials) acc.add(sd.mom_pivot, x, px, y, py, t, pt);
                }
            }
            if (partials) {
                double* red = reinterpret_cast<double*>(smem + pl.red_off);
                hb_block_reduce_moments(acc, red, partials + blockIdx.x, tid, 128, 2);
            }
        }
    } else if (warp < 12) {
        // ===================================================== epilogue warps (hidden output): D[b] -> global scratch
        if (!ly.last) {
            const int wq = warp & 3;
            const int grp = (warp - 4) >> 2;          // 32-column half of every 64-column slab
            const int row = 32 * wq + lane;
            const int te = tid - 128;                 // 0..255 inside the epilogue group
            const uint32_t sw = (uint32_t)(row & 7);
            const uint32_t tlane = tmem_base + ((uint32_t)(32 * wq) << 16) + (uint32_t)(grp * 32);
            const float slope = sd.prelu[ly.layer];
            uint32_t ph_d = 0;                        // bit b: parity of the next completion of D_FULL[b]
            uint32_t jj = 0;                          // staging slabs written so far (2 buffers)
            for (size_t g = cluster_id; g < ngroups; g += nclusters) {
                unsigned char* o_tile = ly.act_out + ((g * CG + rank) * (size_t)NS) * A_SLAB_BYTES;
                for (int nb = 0; nb < NB; ++nb) {
                    const uint32_t b = (uint32_t)nb & 1u;
                    mbar_wait<true>(bar(Q_D_FULL + b), (ph_d >> b) & 1);
                    ph_d ^= 1u << b;
                    tc_fence_after();
                    const int nj = blk_w(nb) >> 6;    // 64-column slabs of this output block
                    uint32_t ra[32], rb[32];
                    tmem_ld32(tlane + b * 256u, ra);
                    for (int j = 0; j < nj; ++j, ++jj) {
                        uint32_t (&cur)[32] = (j & 1) ? rb : ra;
                        uint32_t (&nxt)[32] = (j & 1) ? ra : rb;
                        tmem_ld_wait();
                        if (j + 1 < nj) tmem_ld32(tlane + b * 256u + 64 * (j + 1), nxt);
                        else {                        // every column of D[b] is in registers: hand it back
                            tc_fence_before();
                            __syncwarp();
                            if (lane == 0) mbar_arrive_cluster(bar(Q_D_FREE + b), 0);
                        }
                        const uint32_t stg = sbase + pl.stage_out_off + (jj & 1) * A_SLAB_BYTES;
                        // the bulk store that last read this staging buffer (two slabs ago) must be done reading
                        if (te == 0) bulk_wait_read<1>();
                        asm volatile("bar.sync 3, 256;" ::: "memory");
                        epi_store_slab<32, ACT, F16>(cur, bias_s + nb * 256 + 64 * j + grp * 32, (uint32_t)(grp * 4), slope,
                                                     stg + row * 128, sw);
                        fence_proxy_async();
                        asm volatile("bar.sync 4, 256;" ::: "memory");
                        if (te == 0) {
                            bulk_s2g(o_tile + (size_t)(nb * 4 + j) * A_SLAB_BYTES, stg, A_SLAB_BYTES);
                            bulk_commit();
                        }
                    }
                }
            }
            if (te == 0) bulk_wait_all();             // the scratch must be complete when the kernel ends
        }
    }
    // ---- teardown
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();
    if (warp == 15) {
        tc_fence_after();
        tmem_dealloc<CG>(tmem_base, 512u);
    }
}

// ------------------------------------------------------------------------------- host: plan, packing, launches
int w_round_up(int v, int m) { return (v + m - 1) / m * m; }

bool make_wplan(int prec, int n_linear, const int* widths, TcwPlan& pl) {
    std::memset(&pl, 0, sizeof pl);
    if (prec != 1 && prec != 2) return false;
    if (n_linear < 2) return false;
    int npad = 0;
    for (int l = 0; l < n_linear - 1; ++l) {
        const int w = w_round_up(widths[l + 1], 64);
        if (l == 0) npad = w;
        else if (w != npad) return false;                            // equal (padded) hidden widths only
    }
    if (npad > 1024) return false;
    pl.npad = npad;
    pl.ns = npad / 64;
    pl.nb = (npad + 255) / 256;
    int off = 0;
    pl.ring_off = off;
    off += W_RING * W_STAGE_BYTES;
    pl.stage_out_off = off;
    off += 2 * A_SLAB_BYTES;
    pl.a0_off = off;
    off += 2 * A0_BYTES;
    pl.bias_off = off;
    off += npad * 4;
    pl.bar_off = off;
    off += w_round_up(8 * Q_COUNT + 8, 16);
    pl.red_off = off;
    off += 4 * HB_NMOM * 8;
    pl.total = off;
    return (size_t)pl.total + 1024 <= SMEM_LIMIT;
}

// bytes of one rank's block sequence of layer l
long long w_layer_rank_bytes(const TcwPlan& pl, int n_linear, int l) {
    const long long half_rows = pl.npad / 2;                  // this rank's rows over all output blocks
    if (l == 0) return half_rows * 32;
    if (l == n_linear - 1) return (long long)pl.ns * 1024;
    return half_rows * 128 * pl.ns;
}

template <int ACT, bool F16>
cudaError_t w_launch_one(const HbParticles& p, size_t n_chunk, const HbSurDev& sd, const TcwPlan& pl, const TcwLayer& ly,
                         double* partials, int grid, bool prepare, cudaStream_t s) {
    const size_t smem = (size_t)pl.total + 1024;
    if (prepare) return cudaFuncSetAttribute(hb_sur_tcw_kernel<ACT, F16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(W_THREADS);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = 2;
    at[0].val.clusterDim.y = 1;
    at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, hb_sur_tcw_kernel<ACT, F16>, p, n_chunk, sd, pl, ly, partials);
}

template <bool F16>
cudaError_t w_launch_act(int act, const HbParticles& p, size_t n_chunk, const HbSurDev& sd, const TcwPlan& pl,
                         const TcwLayer& ly, double* partials, int grid, bool prepare, cudaStream_t s) {
    switch (act) {
    case 0: return w_launch_one<0, F16>(p, n_chunk, sd, pl, ly, partials, grid, prepare, s);
    case 1: return w_launch_one<1, F16>(p, n_chunk, sd, pl, ly, partials, grid, prepare, s);
    case 2: return w_launch_one<2, F16>(p, n_chunk, sd, pl, ly, partials, grid, prepare, s);
    default: return w_launch_one<3, F16>(p, n_chunk, sd, pl, ly, partials, grid, prepare, s);
    }
}

}  // namespace

bool hb_tcw_supported(int prec, int n_linear, const int* widths) {
    TcwPlan pl;
    return make_wplan(prec, n_linear, widths, pl);
}

size_t hb_tcw_scratch_bytes(int n_linear, const int* widths) {     // both activation buffers of one chunk
    TcwPlan pl;
    if (!make_wplan(1, n_linear, widths, pl)) return 0;
    return 2 * (size_t)HB_TCW_CHUNK * (size_t)pl.npad * 2;
}

// Image = per layer [rank 0 block sequence | rank 1 block sequence]; off_bytes[l] = start of layer l.
//   layer 0   : per output block nb, this CTA's 128 rows x 32 B, K = 16 no-swizzle (hi | lo copies of W_0)
//   hidden l  : per (nb, s), 128 rows x 128 B swizzled; CTA `rank` holds the rows of neurons nb*256 + rank*128 + i
//   last      : per K slab s, 8 rows x 128 B swizzled (rank 0: outputs 0..7)
size_t hb_tcw_pack_weights(int prec, int n_linear, const int* widths, const float* const* W, void* dst,
                           long long* off_bytes, int* kpad, int* npad) {
    TcwPlan pl;
    if (!make_wplan(prec, n_linear, widths, pl)) return 0;
    size_t total = 0;
    for (int l = 0; l < n_linear; ++l) {
        off_bytes[l] = (long long)total;
        total += 2 * (size_t)w_layer_rank_bytes(pl, n_linear, l);
        npad[l] = l == n_linear - 1 ? 16 : pl.npad;
        kpad[l] = l == 0 ? 16 : pl.npad;
    }
    if (!dst) return total;
    std::memset(dst, 0, total);
    unsigned char* base = static_cast<unsigned char*>(dst);
    auto put = [&](size_t byte, float w) {
        unsigned short bits;
        if (prec == 2) { __half h = __float2half_rn(w); std::memcpy(&bits, &h, 2); }
        else { __nv_bfloat16 h = __float2bfloat16_rn(w); std::memcpy(&bits, &h, 2); }
        std::memcpy(base + byte, &bits, 2);
    };
    for (int l = 0; l < n_linear; ++l) {
        const long long rb = w_layer_rank_bytes(pl, n_linear, l);
        const int fin = widths[l], fout = widths[l + 1];
        for (int rank = 0; rank < 2; ++rank) {
            const size_t r0 = (size_t)off_bytes[l] + (size_t)rank * (size_t)rb;
            if (l == 0) {
                for (int nb = 0; nb < pl.nb; ++nb) {
                    const int hw = std::min(256, pl.npad - 256 * nb) / 2;     // this rank's rows of the block
                    for (int i = 0; i < hw; ++i) {
                        const int o = nb * 256 + rank * hw + i;
                        if (o >= fout) continue;
                        for (int k = 0; k < 12; ++k)
                            put(r0 + (size_t)nb * 4096 + (size_t)(i / 8) * 256 + (size_t)(k / 8) * 128 + (size_t)(i % 8) * 16 + (size_t)(k % 8) * 2,
                                W[0][(size_t)o * fin + (k % 6)]);
                    }
                }
            } else if (l == n_linear - 1) {
                for (int i = 0; i < 8; ++i) {
                    const int o = rank * 8 + i;
                    if (o >= fout) continue;
                    for (int k = 0; k < fin; ++k) {
                        const int s = k / 64, kk = k % 64;
                        put(r0 + (size_t)s * 1024 + (size_t)i * 128 + (size_t)(((kk / 8) ^ (i & 7)) << 4) + (size_t)(kk % 8) * 2,
                            W[l][(size_t)o * fin + k]);
                    }
                }
            } else {
                for (int nb = 0; nb < pl.nb; ++nb) {
                    const int hw = std::min(256, pl.npad - 256 * nb) / 2;
                    for (int s = 0; s < pl.ns; ++s) {
                        const size_t b0 = r0 + (size_t)nb * pl.ns * 16384 + (size_t)s * hw * 128;
                        for (int i = 0; i < hw; ++i) {
                            const int o = nb * 256 + rank * hw + i;
                            if (o >= fout) continue;
                            for (int kk = 0; kk < 64; ++kk) {
                                const int k = s * 64 + kk;
                                if (k >= fin) break;
                                put(b0 + (size_t)i * 128 + (size_t)(((kk / 8) ^ (i & 7)) << 4) + (size_t)(kk % 8) * 2,
                                    W[l][(size_t)o * fin + k]);
                            }
                        }
                    }
                }
            }
        }
    }
    return total;
}

// One surrogate stage = chunks x n_linear launches.  partials: this stage's partial buffer (moment-major rows);
// every chunk's last-layer launch writes its own row range; *nblocks_out = rows the finalize has to sum.
cudaError_t hb_launch_sur_tcw(const HbParticles& p, size_t n, const HbSurDev& sd, double* partials, bool partials_zeroed,
                              int* nblocks_out, int sm_count, bool prepare, cudaStream_t s) {
    TcwPlan pl;
    if (!make_wplan(sd.prec, sd.n_linear, sd.widths, pl)) return cudaErrorNotSupported;
    if (prepare) {
        TcwLayer ly{};
        return sd.prec == 2 ? w_launch_act<true>(sd.act, p, 0, sd, pl, ly, nullptr, 2, true, s)
                            : w_launch_act<false>(sd.act, p, 0, sd, pl, ly, nullptr, 2, true, s);
    }
    if (!sd.act_scratch) return cudaErrorInvalidValue;
    const int grid_max = (sm_count / 2) * 2;
    const size_t nchunks = (n + HB_TCW_CHUNK - 1) / HB_TCW_CHUNK;
    // rows of the partial buffer this stage may write: the whole buffer, or (hb_push_host: partials_zeroed) the row
    // range of one host chunk
    const size_t max_rows = partials_zeroed ? (size_t)HB_MOM_GRID_MAX : (size_t)HB_MOM_MAX_BLOCKS;
    if (partials && nchunks * (size_t)grid_max > max_rows) return cudaErrorNotSupported;
    cudaError_t e = cudaSuccess;
    if (partials && !partials_zeroed)
        e = cudaMemsetAsync(partials, 0, (size_t)HB_NMOM * HB_MOM_MAX_BLOCKS * sizeof(double), s);
    unsigned char* act[2] = {sd.act_scratch, sd.act_scratch + (size_t)HB_TCW_CHUNK * (size_t)pl.npad * 2};
    const int L = sd.n_linear;
    for (size_t c = 0; c < nchunks && e == cudaSuccess; ++c) {
        const size_t off = c * (size_t)HB_TCW_CHUNK;
        const size_t nc = n - off < (size_t)HB_TCW_CHUNK ? n - off : (size_t)HB_TCW_CHUNK;
        const size_t ngroups = ((nc + TILE_M - 1) / TILE_M + 1) / 2;
        size_t clusters = (size_t)(sm_count / 2);
        if (clusters > ngroups) clusters = ngroups;
        const int grid = (int)clusters * 2;
        for (int l = 0; l < L && e == cudaSuccess; ++l) {
            TcwLayer ly;
            ly.first = l == 0;
            ly.last = l == L - 1;
            ly.layer = l;
            ly.w_off = sd.wtc_off[l];
            ly.w_rank_bytes = w_layer_rank_bytes(pl, L, l);
            ly.act_in = act[(l + 1) & 1];
            ly.act_out = act[l & 1];
            ly.row_off = off;
            double* part = (partials && ly.last) ? partials + c * (size_t)grid_max : nullptr;
            e = sd.prec == 2 ? w_launch_act<true>(sd.act, p, nc, sd, pl, ly, part, grid, false, s)
                             : w_launch_act<false>(sd.act, p, nc, sd, pl, ly, part, grid, false, s);
        }
    }
    if (nblocks_out) *nblocks_out = (int)(nchunks * (size_t)grid_max);
    return e;
}
