// hb_mma_rate.cu -- micro-benchmark behind the design of the resident tensor-core kernels: what a
// tcgen05.mma costs to EXECUTE and to ISSUE on this device.  A standalone program (not part of libhb.so):
//     nvcc -gencode arch=compute_100a,code=sm_100a -O3 -std=c++17 -o hb_mma_rate paper_2402_17248_b200/csrc/microbench/hb_mma_rate.cu
//     ./hb_mma_rate
// One CTA pair (or CTA) per SM pair issues 2048 MMAs (kind::f16, K = 16, M = 128 per CTA) and times them with clock64:
//   * N = 16 / 64 / 128 / 256, A from tensor memory ("TS") or shared memory ("SS"), with and without eight epilogue-like
//     warps doing tcgen05.ld / cvt / tcgen05.st on other columns all the while;
//   * the shape of the issuing loop: a tight loop of MMAs against the same loop with a barrier probe or a wait in it
//     (VAR 1-4), and the last layer's pattern (groups of 16 MMAs of N = 16, commit, wait).
// Results of this program on B200: profiles/r2_mma_rate.md.
#include "../hb_tc_common.cuh"
#include <vector>

template <int CG, int VAR>
__global__ void __launch_bounds__(384, 1)
rate_kernel(int N, int ss, int reps, int epi, int rnd, long long* out) {
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    unsigned char* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    const uint32_t sbase = smem_u32(smem);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const uint32_t rank = CG == 1 ? 0u : cluster_rank();
    // layout: [0, 64K) B slabs (4 x 16 KB max: 128 rows x 128 B each for N/CG <= 128 ... 256 rows -> 32 KB per slab: use 128 KB)
    const uint32_t b_off = 0, a_off = 128 * 1024, bar_off = 128 * 1024 + 64 * 1024;
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + bar_off + 64);
    volatile int* done = reinterpret_cast<volatile int*>(smem + bar_off + 128);
    const uint32_t bar = sbase + bar_off;
    for (int i = tid; i < (192 * 1024) / 4; i += blockDim.x) {
        uint32_t h = (uint32_t)i * 2654435761u + blockIdx.x * 40503u;
        h ^= h >> 15; h *= 2246822519u; h ^= h >> 13;
        // two f16 values in [-2, 2): sign random, exponent 0x3c/0x3b.., mantissa random
        const uint32_t lo = (h & 0x83ffu) | 0x3800u, hi = ((h >> 16) & 0x83ffu) | 0x3800u;
        reinterpret_cast<uint32_t*>(smem)[i] = rnd ? (lo | (hi << 16)) : 0u;
    }
    if (tid == 0) {
        mbar_init(bar, 1);
        mbar_init(bar + 8, 1);
        *done = 0;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    fence_proxy_async();
    if (warp == 0) {
        tmem_alloc<CG>(smem_u32(tmem_slot), 512);
        tmem_relinquish<CG>();
    }
    tc_fence_before();
    __syncthreads();
    if (CG == 2) cluster_sync_all();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;
    if (warp < 4) {      // fill the A columns [256, 384) of this lane quarter
        uint32_t q[16];
        for (int c = 0; c < 8; ++c) {
#pragma unroll
            for (int k = 0; k < 16; ++k) {
                uint32_t h = (uint32_t)(tid * 131 + c * 16 + k) * 2654435761u;
                h ^= h >> 15; h *= 2246822519u; h ^= h >> 13;
                q[k] = rnd ? (((h & 0x83ffu) | 0x3800u) | ((((h >> 16) & 0x83ffu) | 0x3800u) << 16)) : 0u;
            }
            tmem_st16(tmem_base + ((uint32_t)(32 * warp) << 16) + 256u + 16u * c, q);
        }
        tmem_st_wait();
        tc_fence_before();
    }
    __syncthreads();
    tc_fence_after();
    if (warp == 0) {
        long long t0 = 0, t1 = 0;
        if (rank == 0) {
            const uint32_t fmt = 0u;   // f16
            const uint32_t idesc = (1u << 4) | (fmt << 7) | (fmt << 10) | ((uint32_t)((TILE_M * CG) >> 4) << 24) | ((uint32_t)(N >> 3) << 17);
            const bool issuer = elect_one();
            const uint64_t bd = make_desc(sbase + b_off);
            const uint64_t ad = make_desc(sbase + a_off);
            const uint64_t bstep = (uint64_t)(((N / CG) * 128) >> 4);
            __syncwarp();
            t0 = clock64();
            if (ss == 10) {
                // the last layer as the kernel issues it: groups of 16 MMAs (K-steps over 128 operand columns, 4 slabs), commit, wait
                uint32_t par = 0;
                for (int r = 0; r < reps / 4; ++r) {
                    if (issuer) {
                        const uint64_t bstep2 = (uint64_t)(((N / CG) * 128) >> 4);
#pragma unroll
                        for (int k = 0; k < 16; ++k)
                            umma_ts<CG, true>(tmem_base + 384, tmem_base + 256 + 8 * k, bd + (uint64_t)(k >> 2) * bstep2 + (uint64_t)(2 * (k & 3)), idesc);
                        umma_commit<CG>(bar);
                    }
                    __syncwarp();
                    mbar_wait<true>(bar, par);
                    par ^= 1;
                    tc_fence_after();
                }
                if (issuer) umma_commit<CG>(bar + 8);
                mbar_wait<false>(bar + 8, 0);
                t1 = clock64();
                *done = 1;
                if (rank == 0 && lane == 0) out[blockIdx.x / CG] = t1 - t0;
                goto finished;
            }
            if (ss >= 2) {
                // kernel-style issue: warp-uniform loop, the elected lane issues inside; ss == 3 adds a completed-barrier probe per slab
                for (int r = 0; r < reps; ++r) {
                    if (VAR == 1) { if (ss == 99) mbar_wait<true>(bar + 8, 1); }          // printf path compiled in, never run
                    if (VAR == 2) { while (!mbar_try(bar + 8, 1)) {} tc_fence_after(); }   // bare try_wait loop on a complete barrier
                    if (VAR == 3) { if (ss == 99) { while (!mbar_try(bar + 8, 1)) {} } }    // bare loop compiled in, never run
                    if (VAR == 4) { mbar_wait<true>(bar + 8, 1); tc_fence_after(); }       // the kernels' wait, on a complete barrier
                    if (issuer) {
                        const uint64_t bj = bd + (uint64_t)(r & 3) * bstep;
                        const uint32_t at = tmem_base + 256 + (uint32_t)(64 * (r & 1));
                        umma_ts<CG, true>(tmem_base, at, bj, idesc);
                        umma_ts<CG, true>(tmem_base, at + 8, bj + 2, idesc);
                        umma_ts<CG, true>(tmem_base, at + 32, bj + 4, idesc);
                        umma_ts<CG, true>(tmem_base, at + 40, bj + 6, idesc);
                    }
                    __syncwarp();
                }
                if (issuer) umma_commit<CG>(bar);
            } else if (issuer) {
                for (int r = 0; r < reps; ++r) {
                    // one "slab": 4 K steps; D at cols [0, N), A (TS) at cols [256, ...)
                    const uint64_t bj = bd + (uint64_t)(r & 3) * bstep;
                    if (ss) {
                        umma<CG, true>(tmem_base, ad, bj, idesc);
                        umma<CG, true>(tmem_base, ad + 2, bj + 2, idesc);
                        umma<CG, true>(tmem_base, ad + 4, bj + 4, idesc);
                        umma<CG, true>(tmem_base, ad + 6, bj + 6, idesc);
                    } else {
                        const uint32_t at = tmem_base + 256 + (uint32_t)(64 * (r & 1));
                        umma_ts<CG, true>(tmem_base, at, bj, idesc);
                        umma_ts<CG, true>(tmem_base, at + 8, bj + 2, idesc);
                        umma_ts<CG, true>(tmem_base, at + 32, bj + 4, idesc);
                        umma_ts<CG, true>(tmem_base, at + 40, bj + 6, idesc);
                    }
                }
                umma_commit<CG>(bar);
            }
            __syncwarp();
        }
        mbar_wait<false>(bar, 0);
        t1 = clock64();
        *done = 1;
        if (rank == 0 && lane == 0) out[blockIdx.x / CG] = t1 - t0;
        finished:;
    } else if (warp >= 4 && epi) {
        // epilogue-like traffic on columns [384, 512): ld 32, cvt, st 16, wait
        const int wq = warp & 3, grp = (warp - 4) >> 2;
        const uint32_t tl = tmem_base + ((uint32_t)(32 * wq) << 16) + 384u + (uint32_t)(grp * 64);
        uint32_t r[32];
        long long cnt = 0;
        while (!*done) {
            tmem_ld32(tl, r);
            tmem_ld_wait();
            if (epi == 2) {
                uint32_t q[16];
#pragma unroll
                for (int k = 0; k < 16; ++k) q[k] = pack2_relu<true>(__uint_as_float(r[2 * k]), __uint_as_float(r[2 * k + 1]));
                tmem_st16(tl + 32, q);
                tmem_st_wait();
            }
            ++cnt;
        }
        if (lane == 0 && blockIdx.x == 0) out[200 + warp] = cnt;
    }
    tc_fence_before();
    __syncthreads();
    if (CG == 2) cluster_sync_all();
    if (warp == 0) {
        tc_fence_after();
        tmem_dealloc<CG>(tmem_base, 512);
    }
}

template <int CG, int VAR>
void run(int N, int ss, int epi, long long* d_out, int rnd = 0) {
    const int reps = 512;
    const size_t smem = 200 * 1024;
    cudaFuncSetAttribute(rate_kernel<CG, VAR>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(148);
    cfg.blockDim = dim3(384);
    cfg.dynamicSmemBytes = smem;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = CG; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    cudaMemset(d_out, 0, 512 * 8);
    for (int it = 0; it < 2; ++it) {
        cudaError_t e = cudaLaunchKernelEx(&cfg, rate_kernel<CG, VAR>, N, ss, reps, epi, rnd, d_out);
        if (e != cudaSuccess) { printf("launch: %s\n", cudaGetErrorString(e)); return; }
        e = cudaDeviceSynchronize();
        if (e != cudaSuccess) { printf("sync: %s\n", cudaGetErrorString(e)); return; }
    }
    std::vector<long long> h(512);
    cudaMemcpy(h.data(), d_out, 512 * 8, cudaMemcpyDeviceToHost);
    double s = 0; long long mx = 0; int nc = 148 / CG;
    for (int i = 0; i < nc; ++i) { s += (double)h[i]; if (h[i] > mx) mx = h[i]; }
    printf("VAR=%d rnd=%d CG=%d N=%3d %s epi=%d : %.1f cycles/MMA (mean over %d clusters), max %.1f ; floor %d ; epi iters warp4 = %lld\n", VAR, rnd, CG, N,
           ss == 0 ? "TS" : (ss == 1 ? "SS" : (ss == 2 ? "TS warp-loop" : "TS groups-of-16")), epi, s / nc / (reps * 4), nc, (double)mx / (reps * 4), 128 * N / 256, h[204]);
}

int main() {
    long long* d_out;
    cudaMalloc(&d_out, 512 * 8);
    printf("-- execution: tight single-thread loop, A from tensor memory (ss=0) / shared memory (ss=1), epilogue traffic off / on\n");
    for (int ss = 0; ss <= 1; ++ss)
        for (int N : {16, 64, 128, 256}) {
            run<2, 0>(N, ss, 0, d_out, 1);
            run<2, 0>(N, ss, 2, d_out, 1);
        }
    for (int N : {128, 256}) run<1, 0>(N, 0, 0, d_out, 1);
    printf("-- issue: warp-uniform loop, elected lane issues 4 MMAs per iteration (VAR 0), + compiled-in but never executed wait (1, 3),\n"
           "   + try_wait on a complete barrier and a fence per iteration (2), + the kernels' mbar_wait and a fence (4)\n");
    for (int N : {16, 128}) {
        run<2, 0>(N, 2, 0, d_out, 1);
        run<2, 1>(N, 2, 0, d_out, 1);
        run<2, 2>(N, 2, 0, d_out, 1);
        run<2, 3>(N, 2, 0, d_out, 1);
        run<2, 4>(N, 2, 0, d_out, 1);
    }
    printf("-- the last layer's pattern: groups of 16 MMAs (16 K steps), commit, wait (ss=10)\n");
    run<2, 0>(16, 10, 0, d_out, 1);
    run<2, 0>(16, 10, 2, d_out, 1);
    return 0;
}
