// hb_epi_cost.cu -- micro-benchmark: what each step of a hidden-layer epilogue event of hb_sur_tc2.cu costs, and what the
// different ways of waiting on an mbarrier cost when the phase completed long ago.  Eight warps per CTA do the step at
// once (two per scheduler, as in the kernel), CTA pairs, one pair per two SMs.  Standalone, not part of libhb.so:
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -std=c++17 --expt-relaxed-constexpr -o hb_epi_cost \
//        paper_2402_17248_b200/csrc/microbench/hb_epi_cost.cu && ./hb_epi_cost       (output: profiles/r2_epi_cost_output.txt)
// The conversion step is measured on values that change every iteration (r ^= iteration), so that it is not hoisted.
#include "../hb_tc_common.cuh"
#include <vector>

template <int O>
__device__ __forceinline__ void ld16o(uint32_t taddr, uint32_t (&r)[64]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
        : "=r"(r[O + 0]), "=r"(r[O + 1]), "=r"(r[O + 2]), "=r"(r[O + 3]), "=r"(r[O + 4]), "=r"(r[O + 5]), "=r"(r[O + 6]),
          "=r"(r[O + 7]), "=r"(r[O + 8]), "=r"(r[O + 9]), "=r"(r[O + 10]), "=r"(r[O + 11]), "=r"(r[O + 12]), "=r"(r[O + 13]),
          "=r"(r[O + 14]), "=r"(r[O + 15])
        : "r"(taddr) : "memory");
}
template <int O>
__device__ __forceinline__ void st8o(uint32_t taddr, const uint32_t (&q)[64]) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
                 ::"r"(taddr), "r"(q[O + 0]), "r"(q[O + 1]), "r"(q[O + 2]), "r"(q[O + 3]), "r"(q[O + 4]), "r"(q[O + 5]),
                   "r"(q[O + 6]), "r"(q[O + 7]) : "memory");
}

// the wait the kernels used until round 2: 16 tries, then a clocked sleep loop whose hang guard prints and traps
__device__ __forceinline__ void wait_printf(uint32_t bar, uint32_t parity) {
#pragma unroll 1
    for (int i = 0; i < 16; ++i)
        if (mbar_try(bar, parity)) return;
    const long long t0 = clock64();
    while (!mbar_try_sleep(bar, parity)) {
        if (clock64() - t0 > 4000000000LL) {
            printf("timeout (block %d thread %d bar %u parity %u)\n", blockIdx.x, threadIdx.x, bar, parity);
            __trap();
        }
    }
}
__device__ __forceinline__ void wait_bare_try(uint32_t bar, uint32_t parity) { while (!mbar_try(bar, parity)) {} }
__device__ __forceinline__ void wait_counter(uint32_t bar, uint32_t parity) {
    uint32_t n = 0;
    while (!mbar_try(bar, parity)) {
        if (++n > 100000000u) __trap();
    }
}

enum : int {
    M_WAIT_PRINTF = 1, M_LD = 2, M_ARRIVE1 = 4, M_CVT = 8, M_ST = 16, M_ARRIVE2 = 32, M_TEST = 64, M_TRY = 128,
    M_FENCE_AFTER = 256, M_WAIT_GUARDED = 512, M_WAIT_SPIN = 1024, M_WAIT_BARE_TRY = 2048, M_WAIT_COUNTER = 4096,
    M_XOR = 8192, M_CVT_PLAIN = 16384, M_CVT_BF16 = 32768, M_CVT_TANH = 65536
};

template <int MASK>
__global__ void __launch_bounds__(448, 1) epi_kernel(int reps, long long* out) {
    extern __shared__ __align__(1024) unsigned char smem[];
    const uint32_t sbase = smem_u32(smem);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + 256);
    const uint32_t bar = sbase;          // bar + 0: its phase 0 is complete; bar + 8, bar + 16: arrival sinks
    if (tid == 0) {
        mbar_init(bar, 1);
        mbar_init(bar + 8, 16);
        mbar_init(bar + 16, 16);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 13) {
        tmem_alloc<2>(smem_u32(tmem_slot), 512);
        tmem_relinquish<2>();
    }
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();
    tc_fence_after();
    if (tid == 0) mbar_arrive_local(bar);
    __syncthreads();
    const uint32_t tmem_base = *tmem_slot;
    if (warp >= 4 && warp < 12) {
        const int wq = warp & 3, grp = (warp - 4) >> 2;
        const uint32_t src = tmem_base + ((uint32_t)(32 * wq) << 16) + 256u + (uint32_t)(grp * 64);
        const uint32_t dst = tmem_base + ((uint32_t)(32 * wq) << 16) + (uint32_t)(grp * 32);
        uint32_t r[64];
#pragma unroll
        for (int i = 0; i < 64; ++i) r[i] = 0x3c003c00u + i;
        __syncwarp();
        const long long t0 = clock64();
        for (int it = 0; it < reps; ++it) {
            if (MASK & M_WAIT_PRINTF) wait_printf(bar, 0);
            if (MASK & M_WAIT_GUARDED) mbar_wait<true>(bar, 0);
            if (MASK & M_WAIT_SPIN) mbar_spin(bar, 0);
            if (MASK & M_WAIT_BARE_TRY) wait_bare_try(bar, 0);
            if (MASK & M_WAIT_COUNTER) wait_counter(bar, 0);
            if (MASK & M_TEST) { if (!mbar_test(bar, 0)) break; }
            if (MASK & M_TRY) { if (!mbar_try(bar, 0)) break; }
            if (MASK & M_FENCE_AFTER) tc_fence_after();
            if (MASK & M_LD) {
                ld16o<0>(src, r);
                ld16o<16>(src + 16u, r);
                ld16o<32>(src + 32u, r);
                ld16o<48>(src + 48u, r);
                tmem_ld_wait();
            }
            if (MASK & M_ARRIVE1) {
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive_cluster(bar + 8, 0);
            }
            if (MASK & M_CVT) {
#pragma unroll
                for (int i = 0; i < 64; ++i) r[i] ^= (uint32_t)it;          // new values every iteration
#pragma unroll
                for (int c = 0; c < 4; ++c)
#pragma unroll
                    for (int k = 0; k < 8; ++k)
                        r[8 * c + k] = act_pack<1, true>(__uint_as_float(r[16 * c + 2 * k]), __uint_as_float(r[16 * c + 2 * k + 1]), 0.f);
            }
            if (MASK & (M_XOR | M_CVT_PLAIN | M_CVT_BF16 | M_CVT_TANH)) {
#pragma unroll
                for (int i = 0; i < 64; ++i) r[i] ^= (uint32_t)it;
            }
            if (MASK & M_CVT_PLAIN) {       // no activation fused into the conversion
#pragma unroll
                for (int c = 0; c < 4; ++c)
#pragma unroll
                    for (int k = 0; k < 8; ++k)
                        r[8 * c + k] = pack2<true>(__uint_as_float(r[16 * c + 2 * k]), __uint_as_float(r[16 * c + 2 * k + 1]));
            }
            if (MASK & M_CVT_BF16) {
#pragma unroll
                for (int c = 0; c < 4; ++c)
#pragma unroll
                    for (int k = 0; k < 8; ++k)
                        r[8 * c + k] = act_pack<1, false>(__uint_as_float(r[16 * c + 2 * k]), __uint_as_float(r[16 * c + 2 * k + 1]), 0.f);
            }
            if (MASK & M_CVT_TANH) {
#pragma unroll
                for (int c = 0; c < 4; ++c)
#pragma unroll
                    for (int k = 0; k < 8; ++k)
                        r[8 * c + k] = act_pack<3, true>(__uint_as_float(r[16 * c + 2 * k]), __uint_as_float(r[16 * c + 2 * k + 1]), 0.f);
            }
            if (MASK & M_ST) {
                st8o<0>(dst, r);
                st8o<8>(dst + 8u, r);
                st8o<16>(dst + 16u, r);
                st8o<24>(dst + 24u, r);
                tmem_st_wait();
            }
            if (MASK & M_ARRIVE2) {
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive_cluster(bar + 16, 0);
            }
        }
        const long long t1 = clock64();
        uint32_t s = 0;
#pragma unroll
        for (int i = 0; i < 64; ++i) s += r[i];
        if (lane == 0 && warp == 4) out[blockIdx.x] = t1 - t0 + (s == 0x12345u ? 1 : 0);
    }
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();
    if (warp == 13) {
        tc_fence_after();
        tmem_dealloc<2>(tmem_base, 512);
    }
}

template <int MASK>
void run(const char* what, long long* d_out) {
    const int reps = 2000;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(148);
    cfg.blockDim = dim3(448);
    cfg.dynamicSmemBytes = 1024;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = 2; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    for (int it = 0; it < 2; ++it) {
        cudaError_t e = cudaLaunchKernelEx(&cfg, epi_kernel<MASK>, reps, d_out);
        if (e != cudaSuccess) { printf("launch: %s\n", cudaGetErrorString(e)); return; }
        e = cudaDeviceSynchronize();
        if (e != cudaSuccess) { printf("sync: %s\n", cudaGetErrorString(e)); return; }
    }
    std::vector<long long> h(148);
    cudaMemcpy(h.data(), d_out, 148 * 8, cudaMemcpyDeviceToHost);
    double s = 0;
    for (int i = 0; i < 148; ++i) s += (double)h[i];
    printf("%-78s %7.1f cycles / iteration\n", what, s / 148 / reps);
}

int main() {
    long long* d_out;
    cudaMalloc(&d_out, 148 * 8);
    printf("waits on a barrier whose phase is complete (8 warps per CTA at once)\n");
    run<M_TEST>("mbarrier.test_wait", d_out);
    run<M_TRY>("mbarrier.try_wait", d_out);
    run<M_WAIT_SPIN>("mbar_spin (the issuers' wait: bare test_wait loop)", d_out);
    run<M_WAIT_BARE_TRY>("bare try_wait loop", d_out);
    run<M_WAIT_COUNTER>("try_wait loop, iteration-count guard, trap", d_out);
    run<M_WAIT_GUARDED>("mbar_wait<true> (every other role: try_wait, clock guard, trap)", d_out);
    run<M_WAIT_PRINTF>("the wait used before: 16 tries, clocked sleep loop, printf + trap inline", d_out);
    run<M_FENCE_AFTER>("tcgen05.fence::after_thread_sync", d_out);
    printf("steps of one epilogue event (64 accumulator columns per warp)\n");
    run<M_LD>("4 x tcgen05.ld.x16 + wait::ld", d_out);
    run<M_ARRIVE1>("fence::before + syncwarp + mbarrier.arrive (cluster)", d_out);
    run<M_XOR>("64 xor (what the next lines add to the conversions so that they are not hoisted)", d_out);
    run<M_CVT>("64 xor + 32 cvt.rn.relu.f16x2", d_out);
    run<M_CVT_PLAIN>("64 xor + 32 cvt.rn.f16x2", d_out);
    run<M_CVT_BF16>("64 xor + 32 cvt.rn.relu.bf16x2", d_out);
    run<M_CVT_TANH>("64 xor + 64 tanh.approx + 32 cvt.rn.f16x2", d_out);
    run<M_ST>("4 x tcgen05.st.x8 + wait::st", d_out);
    run<M_LD | M_CVT | M_ST>("ld + cvt + st", d_out);
    run<M_WAIT_GUARDED | M_FENCE_AFTER | M_LD | M_ARRIVE1 | M_CVT | M_ST | M_ARRIVE2>("whole event, guarded wait", d_out);
    run<M_WAIT_PRINTF | M_FENCE_AFTER | M_LD | M_ARRIVE1 | M_CVT | M_ST | M_ARRIVE2>("whole event, the wait used before", d_out);
    return 0;
}
