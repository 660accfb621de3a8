// hb_sur_tc2.cu -- tensor-core surrogate stage (rows a4-a6), weights resident in shared memory, TWO tiles in
// flight per CTA pair.  Chosen for nets whose pair plan leaves room for an operand ring (C3: 6-256^3-6).
//
// hb_sur_tc.cu keeps one tile in flight and pays, once per layer, the latency between "accumulator complete" and
// "first slab of the next operand visible to the MMA issuer" (~900 cycles of an idle tensor pipe against 2048 cycles
// of MMAs, profiles/r1_kernels_v2.md).  Here the CTA pair owns two tile slots X and Y, each with its own TMEM
// accumulator (2 x 256 columns), and the MMA issuer alternates  X.L0 Y.L0 X.L1 Y.L1 ...: while the epilogue warps
// turn D_X of layer l into the layer l+1 operand of X, the tensor pipe runs layer l of Y.  The operands live in a
// FIFO ring of 16 KB K slabs (64 inputs x 128 particles): produced by the epilogue warps in exactly the order the
// MMA issuer consumes them; a slab is handed back by a tcgen05.commit on its RING_EMPTY barrier.  With the weights
// (136 KB per CTA for C3) the ring has five slots, one more than a layer needs, so the producer runs one slab ahead
// of the MMAs that free its slots.
// Warp roles (14 warps): 0-3 IO (a4 prologue straight from global memory, a6 output, a3 moments), 4-11 hidden-layer
// epilogue, 12 weight loader (TMA bulk copies, once), 13 MMA issuer (leader CTA, elected lane).
#include "hb_tc_common.cuh"

namespace {

constexpr int T2_THREADS = 448;
constexpr int T2_MAX_RING = 8;
enum : int {
    T_W = 0,              // weights resident (local)
    T_A0_FULL = 1,        // [2] layer-0 operand of slot s written (leader; 4 IO warps x 2 CTAs)
    T_A0_FREE = 3,        // [2] layer-0 MMA of slot s complete: its operand buffer may be rewritten (both, commit)
    T_RING_FULL = 5,      // [8] ring slab written (leader; 8 epilogue warps x 2 CTAs)
    T_RING_EMPTY = 13,    // [8] ring slab consumed (both, commit)
    T_D_FULL = 21,        // [2] accumulator of slot s complete, hidden layer (both, commit)
    T_D_LAST = 23,        // [2] accumulator of slot s complete, last layer (both, commit)
    T_OUT_READ = 25,      // [2] last layer's accumulator of slot s read by the IO warps (leader; 4 x 2)
    T_COUNT = 27
};

struct Tc2Plan {
    int n_linear;
    int nslab[HB_MAX_LINEAR];         // 64-wide K slabs of layer l's operand (layer 0: 0)
    int npad[HB_MAX_LINEAR];          // padded fan-out (both CTAs)
    int w_off[HB_MAX_LINEAR];         // smem byte offset of layer l's weights (this CTA's rows)
    int w_slab_bytes[HB_MAX_LINEAR];  // l >= 1: (npad / 2) * 128;  l = 0: (npad / 2) * 32
    int ring;                         // ring slots
    int a_off, a0_off, bar_off, red_off, total;
    int w_bytes_total;
};

template <int ACT, bool F16>
__global__ void __launch_bounds__(T2_THREADS, 1)
hb_sur_tc2_kernel(HbParticles p, size_t n, const __grid_constant__ HbSurDev sd, const __grid_constant__ Tc2Plan pl,
                  double* __restrict__ partials) {
    constexpr int CG = 2;
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    unsigned char* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    const uint32_t sbase = smem_u32(smem);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const uint32_t rank = cluster_rank();
    const size_t ntiles = (n + TILE_M - 1) / TILE_M;
    const size_t ngroups = (ntiles + CG - 1) / CG;
    const size_t cluster_id = blockIdx.x / CG, nclusters = gridDim.x / CG;
    // tiles (groups of 2 x 128 particles) of this CTA pair: g_k = cluster_id + k * nclusters, k < nk; slot = k & 1
    const size_t nk = cluster_id < ngroups ? (ngroups - cluster_id + nclusters - 1) / nclusters : 0;
    const int L = pl.n_linear, R = pl.ring;

    const uint32_t bar0 = sbase + pl.bar_off;
    auto bar = [&](int i) -> uint32_t { return bar0 + 8u * (uint32_t)i; };
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + pl.bar_off + 8 * T_COUNT);

    if (tid == 0) {
        mbar_init(bar(T_W), 1);
        for (int s = 0; s < 2; ++s) {
            mbar_init(bar(T_A0_FULL + s), 4 * CG);
            mbar_init(bar(T_A0_FREE + s), 1);
            mbar_init(bar(T_D_FULL + s), 1);
            mbar_init(bar(T_D_LAST + s), 1);
            mbar_init(bar(T_OUT_READ + s), 4 * CG);
        }
        for (int r = 0; r < T2_MAX_RING; ++r) {
            mbar_init(bar(T_RING_FULL + r), 8 * CG);
            mbar_init(bar(T_RING_EMPTY + r), 1);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 13) {
        tmem_alloc<CG>(smem_u32(tmem_slot), 512u);
        tmem_relinquish<CG>();
    }
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    if (warp == 12) {
        // ===================================================== weight loader (once)
        if (lane == 0) {
            mbar_expect_tx(bar(T_W), (uint32_t)pl.w_bytes_total);
            const unsigned char* wg = reinterpret_cast<const unsigned char*>(sd.wtc);
            bulk_g2s(sbase + pl.w_off[0], wg + sd.wtc_off[0] + (size_t)rank * pl.w_slab_bytes[0],
                     (uint32_t)pl.w_slab_bytes[0], bar(T_W));
            for (int l = 1; l < L; ++l)
                for (int s = 0; s < pl.nslab[l]; ++s) {
                    const unsigned char* src = wg + sd.wtc_off[l] + (size_t)s * pl.npad[l] * 128 + (size_t)rank * pl.w_slab_bytes[l];
                    bulk_g2s(sbase + pl.w_off[l] + s * pl.w_slab_bytes[l], src, (uint32_t)pl.w_slab_bytes[l], bar(T_W));
                }
        }
        __syncwarp();
    } else if (warp == 13) {
        // ===================================================== MMA issuer (leader CTA): X.L0 Y.L0 X.L1 Y.L1 ...
        if (rank == 0) {
            const uint32_t fmt = F16 ? 0u : 1u;
            const uint32_t idesc_base = (1u << 4) | (fmt << 7) | (fmt << 10) | ((uint32_t)((TILE_M * CG) >> 4) << 24);
            const bool issuer = elect_one();
            const uint64_t a_desc0 = make_desc(sbase + pl.a_off);
            const uint64_t w0_desc = make_desc_l0(sbase + pl.w_off[0]);
            uint32_t rc = 0, phc = 0;                // ring consumer position and phase
            for (size_t k0 = 0; k0 < nk; k0 += 2) {
                const uint32_t q = (uint32_t)(k0 >> 1);                 // use count of a slot so far
                for (int l = 0; l < L; ++l) {
                    const uint32_t idesc = idesc_base | ((uint32_t)(pl.npad[l] >> 3) << 17);
                    const int nsl = pl.nslab[l];
                    const uint64_t bd = l ? make_desc(sbase + pl.w_off[l]) : 0ull;
                    const uint64_t bd_step = (uint64_t)(pl.w_slab_bytes[l] >> 4);
                    for (uint32_t s = 0; s < 2; ++s) {
                        if (k0 + s >= nk) break;
                        const uint32_t d_tmem = tmem_base + s * 256u;
                        const bool last = l == L - 1;
                        if (l == 0) {
                            // D[s] still holds the outputs of the slot's previous tile until the IO warps read them
                            if (q > 0) mbar_wait<true>(bar(T_OUT_READ + s), (q - 1) & 1);
                            mbar_wait<true>(bar(T_A0_FULL + s), q & 1);
                            tc_fence_after();
                            if (issuer) {
                                umma<CG, false>(d_tmem, make_desc_l0(sbase + pl.a0_off + s * A0_BYTES), w0_desc, idesc);
                                umma_commit<CG>(bar(T_A0_FREE + s));
                                umma_commit<CG>(last ? bar(T_D_LAST + s) : bar(T_D_FULL + s));
                            }
                        } else {
                            // the first MMA overwrites D[s]: the slot's previous epilogue must have written its last
                            // slab (slabs complete in ring order, so the earlier ones are complete too)
                            uint32_t rl = rc + (uint32_t)nsl - 1, phl = phc;
                            if (rl >= (uint32_t)R) { rl -= R; phl ^= 1; }
                            mbar_wait<true>(bar(T_RING_FULL + rl), phl);
                            tc_fence_after();
                            for (int j = 0; j < nsl; ++j) {
                                if (issuer) {
                                    const uint64_t ad = a_desc0 + (uint64_t)(rc * (A_SLAB_BYTES >> 4));
                                    const uint64_t bj = bd + (uint64_t)j * bd_step;
                                    if (j == 0) umma<CG, false>(d_tmem, ad, bj, idesc);
                                    else umma<CG, true>(d_tmem, ad, bj, idesc);
                                    umma<CG, true>(d_tmem, ad + 2, bj + 2, idesc);
                                    umma<CG, true>(d_tmem, ad + 4, bj + 4, idesc);
                                    umma<CG, true>(d_tmem, ad + 6, bj + 6, idesc);
                                    umma_commit<CG>(bar(T_RING_EMPTY + rc));
                                }
                                if (++rc == (uint32_t)R) { rc = 0; phc ^= 1; }
                            }
                            if (issuer) umma_commit<CG>(last ? bar(T_D_LAST + s) : bar(T_D_FULL + s));
                        }
                        __syncwarp();
                    }
                }
            }
        }
        __syncwarp();
    } else if (warp < 4) {
        // ===================================================== IO warps: prologue of tile k+2, output of tile k
        const int row = 32 * warp + lane;        // tile row = TMEM lane = particle within the tile
        const uint32_t a0_row = sbase + pl.a0_off + (uint32_t)(row >> 3) * 256 + (uint32_t)(row & 7) * 16;
        const uint32_t tlane = tmem_base + ((uint32_t)(32 * warp) << 16);
        float bl[6];
#pragma unroll
        for (int j = 0; j < 6; ++j) bl[j] = sd.btc[sd.btc_off[L - 1] + j];
        HbMomAcc acc;
        acc.clear();
        // a4: load (coalesced: a warp reads 128 consecutive bytes per coordinate), convert, normalise, split,
        // write the layer-0 operand of tile k into its slot's buffer
        auto prologue = [&](size_t k) {
            const uint32_t s = (uint32_t)(k & 1);
            const size_t tile = (cluster_id + k * nclusters) * CG + rank;
            const size_t i = tile * TILE_M + row;
            const bool valid = tile < ntiles && i < n;
            float c[6] = {0, 0, 0, 0, 0, 0};
            if (valid) {
#pragma unroll
                for (int j = 0; j < 6; ++j) c[j] = __ldcs(p.v[j] + i);
            }
            uint32_t q0[4], q1[4];
            tc_make_a0_row<F16>(sd, valid, c, q0, q1);
            const uint32_t dst = a0_row + s * A0_BYTES;
            sts128(dst, q0);
            sts128(dst + 128, q1);
            fence_proxy_async();
            __syncwarp();
            if (lane == 0) mbar_arrive_cluster(bar(T_A0_FULL + s), 0);
        };
        mbar_wait<false>(bar(T_W), 0);           // this CTA's weights are resident before the first MMA may start
        if (nk > 0) prologue(0);
        if (nk > 1) prologue(1);
        for (size_t k = 0; k < nk; ++k) {
            const uint32_t s = (uint32_t)(k & 1), par = (uint32_t)((k >> 1) & 1);
            if (k + 2 < nk) {
                mbar_wait<false>(bar(T_A0_FREE + s), par);      // layer 0 of tile k has read the slot's buffer
                prologue(k + 2);
            }
            const size_t tile = (cluster_id + k * nclusters) * CG + rank;
            const size_t i = tile * TILE_M + row;
            const bool valid = tile < ntiles && i < n;
            mbar_wait<false>(bar(T_D_LAST + s), par);
            tc_fence_after();
            uint32_t r[8];
            tmem_ld8(tlane + s * 256u, r);
            tmem_ld_wait();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive_cluster(bar(T_OUT_READ + s), 0);
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
        // ===================================================== hidden-layer epilogue warps: X.0 Y.0 X.1 Y.1 ...
        const int wq = warp & 3;
        const int grp = (warp - 4) >> 2;          // 32-column half of every 64-column slab
        const int row = 32 * wq + lane;
        const uint32_t ring_row = sbase + pl.a_off + row * 128;
        const uint32_t sw = (uint32_t)(row & 7);
        const uint32_t tlane = tmem_base + ((uint32_t)(32 * wq) << 16) + (uint32_t)(grp * 32);
        uint32_t ph_d = 0;                        // bit s: parity of the next completion of D_FULL[s]
        uint32_t rp = 0, php = 0;                 // ring producer position and phase
        for (size_t k0 = 0; k0 < nk; k0 += 2) {
            for (int l = 0; l < L - 1; ++l) {
                const int nsl = pl.npad[l] >> 6;
                const float* bl = sd.btc + sd.btc_off[l] + grp * 32;     // biases from global memory (L1-resident)
                const float slope = sd.prelu[l];
                for (uint32_t s = 0; s < 2; ++s) {
                    if (k0 + s >= nk) break;
                    const uint32_t t0 = tlane + s * 256u;
                    mbar_wait<true>(bar(T_D_FULL + s), (ph_d >> s) & 1);
                    ph_d ^= 1u << s;
                    tc_fence_after();
                    uint32_t ra[32], rb[32];
                    tmem_ld32(t0, ra);
                    for (int j = 0; j < nsl; j += 2) {
                        tmem_ld_wait();
                        if (j + 1 < nsl) tmem_ld32(t0 + 64 * (j + 1), rb);
                        mbar_wait<true>(bar(T_RING_EMPTY + rp), php ^ 1);
                        epi_store_slab<32, ACT, F16>(ra, bl + 64 * j, (uint32_t)(grp * 4), slope, ring_row + rp * A_SLAB_BYTES, sw);
                        fence_proxy_async();
                        tc_fence_before();
                        __syncwarp();
                        if (lane == 0) mbar_arrive_cluster(bar(T_RING_FULL + rp), 0);
                        if (++rp == (uint32_t)R) { rp = 0; php ^= 1; }
                        if (j + 1 < nsl) {
                            tmem_ld_wait();
                            if (j + 2 < nsl) tmem_ld32(t0 + 64 * (j + 2), ra);
                            mbar_wait<true>(bar(T_RING_EMPTY + rp), php ^ 1);
                            epi_store_slab<32, ACT, F16>(rb, bl + 64 * (j + 1), (uint32_t)(grp * 4), slope, ring_row + rp * A_SLAB_BYTES, sw);
                            fence_proxy_async();
                            tc_fence_before();
                            __syncwarp();
                            if (lane == 0) mbar_arrive_cluster(bar(T_RING_FULL + rp), 0);
                            if (++rp == (uint32_t)R) { rp = 0; php ^= 1; }
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
    if (warp == 13) {
        tc_fence_after();
        tmem_dealloc<CG>(tmem_base, 512u);
    }
}

// ------------------------------------------------------------------------------- host: plan + launch
int t2_round_up(int v, int m) { return (v + m - 1) / m * m; }

// Same operand geometry and weight image as hb_sur_tc.cu's CTA-pair plan (hb_tc_pack_weights).
bool make_plan2(int n_linear, const int* widths, Tc2Plan& pl) {
    std::memset(&pl, 0, sizeof pl);
    if (n_linear < 2) return false;
    pl.n_linear = n_linear;
    int off = 0, maxslab = 0, maxn = 0;
    for (int l = 0; l < n_linear; ++l) {
        const bool last = l == n_linear - 1;
        pl.npad[l] = last ? 16 : t2_round_up(widths[l + 1], 64);
        pl.nslab[l] = l == 0 ? 0 : pl.npad[l - 1] / 64;
        if ((pl.npad[l] / 2) % 8) return false;
        pl.w_slab_bytes[l] = pl.npad[l] / 2 * (l == 0 ? 32 : 128);
        pl.w_off[l] = off;
        off += (l == 0 ? 1 : pl.nslab[l]) * pl.w_slab_bytes[l];
        pl.w_bytes_total += (l == 0 ? 1 : pl.nslab[l]) * pl.w_slab_bytes[l];
        off = t2_round_up(off, 1024);
        if (pl.nslab[l] > maxslab) maxslab = pl.nslab[l];
        if (pl.npad[l] > maxn) maxn = pl.npad[l];
    }
    if (maxn > 256) return false;                                   // two accumulators in 512 TMEM columns
    pl.a_off = off;
    const int fixed = 2 * A0_BYTES + t2_round_up(8 * T_COUNT + 8, 16) + 4 * HB_NMOM * 8 + 1024;
    int ring = ((int)SMEM_LIMIT - off - fixed) / A_SLAB_BYTES;
    if (ring > T2_MAX_RING) ring = T2_MAX_RING;
    if (ring < maxslab + 1) return false;                           // one slab of run-ahead at least
    pl.ring = ring;
    off += ring * A_SLAB_BYTES;
    pl.a0_off = off;
    off += 2 * A0_BYTES;
    pl.bar_off = off;
    off += t2_round_up(8 * T_COUNT + 8, 16);
    pl.red_off = off;
    off += 4 * HB_NMOM * 8;
    pl.total = off;
    return (size_t)pl.total + 1024 <= SMEM_LIMIT;
}

template <int ACT, bool F16>
cudaError_t t2_launch_one(const HbParticles& p, size_t n, const HbSurDev& sd, const Tc2Plan& pl, double* partials, int grid,
                          cudaStream_t s) {
    const size_t smem = (size_t)pl.total + 1024;
    cudaError_t e = cudaFuncSetAttribute(hb_sur_tc2_kernel<ACT, F16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(T2_THREADS);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = 2;
    at[0].val.clusterDim.y = 1;
    at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, hb_sur_tc2_kernel<ACT, F16>, p, n, sd, pl, partials);
}

template <bool F16>
cudaError_t t2_launch_act(const HbParticles& p, size_t n, const HbSurDev& sd, const Tc2Plan& pl, double* partials, int grid,
                          cudaStream_t s) {
    switch (sd.act) {
    case 0: return t2_launch_one<0, F16>(p, n, sd, pl, partials, grid, s);
    case 1: return t2_launch_one<1, F16>(p, n, sd, pl, partials, grid, s);
    case 2: return t2_launch_one<2, F16>(p, n, sd, pl, partials, grid, s);
    default: return t2_launch_one<3, F16>(p, n, sd, pl, partials, grid, s);
    }
}

}  // namespace

bool hb_tc2_supported(int n_linear, const int* widths) {
    Tc2Plan pl;
    return make_plan2(n_linear, widths, pl);
}

cudaError_t hb_launch_sur_tc2(const HbParticles& p, size_t n, const HbSurDev& sd, double* partials, int* nblocks_out,
                              int sm_count, cudaStream_t s) {
    Tc2Plan pl;
    if (!make_plan2(sd.n_linear, sd.widths, pl)) return cudaErrorNotSupported;
    const size_t ntiles = (n + TILE_M - 1) / TILE_M;
    const size_t ngroups = (ntiles + 1) / 2;
    size_t clusters = (size_t)(sm_count / 2);
    if (clusters > ngroups) clusters = ngroups;
    if (clusters < 1) clusters = 1;
    const int grid = (int)clusters * 2;
    if (nblocks_out) *nblocks_out = grid;
    return sd.prec == 2 ? t2_launch_act<true>(p, n, sd, pl, partials, grid, s) : t2_launch_act<false>(p, n, sd, pl, partials, grid, s);
}
