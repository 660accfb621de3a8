// hb_peaks.cu -- hb_device_peaks(): measured throughput of the pipes libhb's kernels are bound by, on the device at
// hand: fp32 FMA, fp64 FMA, MUFU tanh, and the tcgen05 tensor pipe for kind::f16 and kind::tf32 operands.  The
// rooflines of the ALU-bound kernels (hb_sur_fp32_kernel, hb_run_sequential_kernel, the tanh stages) and of the tf32
// mode are quoted against these numbers instead of datasheet unit counts (bench.py).  Short kernels (a few
// milliseconds each): burst rates at the clock the device runs unloaded, not a sustained, power-limited figure.
#include "../../include/hb.h"
#include "hb_tc_common.cuh"

namespace {

constexpr int PK_THREADS = 256;

// `iters` rounds of 8 independent chains per thread
__global__ void __launch_bounds__(PK_THREADS) pk_ffma_kernel(float* out, int iters, float a, float b) {
    float v[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) v[i] = (float)(threadIdx.x + i);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) v[i] = fmaf(v[i], a, b);
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += v[i];
    if (s == 123.456f) out[0] = s;          // never true: keeps the chains alive
}
__global__ void __launch_bounds__(PK_THREADS) pk_dfma_kernel(double* out, int iters, double a, double b) {
    double v[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) v[i] = (double)(threadIdx.x + i);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) v[i] = fma(v[i], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += v[i];
    if (s == 123.456) out[0] = s;
}
__global__ void __launch_bounds__(PK_THREADS) pk_tanh_kernel(float* out, int iters) {
    float v[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) v[i] = 0.01f * (float)(threadIdx.x + i);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) v[i] = hb_tanh_approx(v[i]);
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += v[i];
    if (s == 123.456f) out[0] = s;
}

// One CTA per SM: `reps` x 4 MMAs of M128 x N256 x K(16 | 8), both operands from shared memory (128-byte swizzle, zeros),
// accumulating into the same 256 TMEM columns.
template <bool T32>
__global__ void __launch_bounds__(128, 1) pk_mma_kernel(int reps) {
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    unsigned char* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    const uint32_t sbase = smem_u32(smem);
    const int tid = threadIdx.x, warp = tid >> 5;
    const uint32_t a_off = 0, b_off = 16 * 1024, bar_off = 48 * 1024;
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + bar_off + 16);
    for (int i = tid; i < (48 * 1024) / 16; i += 128) reinterpret_cast<uint4*>(smem)[i] = make_uint4(0, 0, 0, 0);
    if (tid == 0) {
        mbar_init(sbase + bar_off, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    fence_proxy_async();
    if (warp == 0) {
        tmem_alloc<1>(smem_u32(tmem_slot), 256);
        tmem_relinquish<1>();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;
    if (warp == 0) {
        // idesc: fp32 accumulate, A/B format f16 (0) or tf32 (2), M = 128, N = 256
        const uint32_t fmt = T32 ? 2u : 0u;
        const uint32_t idesc = (1u << 4) | (fmt << 7) | (fmt << 10) | ((uint32_t)(TILE_M >> 4) << 24) | ((uint32_t)(256 >> 3) << 17);
        const uint64_t ad = make_desc(sbase + a_off), bd = make_desc(sbase + b_off);
        if (elect_one()) {
            for (int r = 0; r < reps; ++r) {
                umma<1, true, T32>(tmem_base, ad, bd, idesc);
                umma<1, true, T32>(tmem_base, ad + 2, bd + 2, idesc);
                umma<1, true, T32>(tmem_base, ad + 4, bd + 4, idesc);
                umma<1, true, T32>(tmem_base, ad + 6, bd + 6, idesc);
            }
            umma_commit<1>(sbase + bar_off);
        }
        __syncwarp();
        mbar_wait<false>(sbase + bar_off, 0);
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) {
        tc_fence_after();
        tmem_dealloc<1>(tmem_base, 256);
    }
}

template <typename F>
cudaError_t time_ms(F launch, float* ms) {
    cudaEvent_t e0, e1;
    cudaError_t e = cudaEventCreate(&e0);
    if (e != cudaSuccess) return e;
    e = cudaEventCreate(&e1);
    if (e != cudaSuccess) return e;
    float best = 1e30f;
    for (int it = 0; it < 4 && e == cudaSuccess; ++it) {          // first round warms up; best of the rest
        cudaEventRecord(e0);
        launch();
        cudaEventRecord(e1);
        e = cudaEventSynchronize(e1);
        if (e == cudaSuccess) e = cudaGetLastError();
        float t = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&t, e0, e1);
        if (it > 0 && t < best) best = t;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    *ms = best;
    return e;
}

}  // namespace

extern "C" hb_status hb_device_peaks(int cuda_device, double* out5) {
    if (!out5) return HB_ERR_INVALID_ARG;
    for (int i = 0; i < 5; ++i) out5[i] = 0.0;
    int ndev = 0, prev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || cuda_device < 0 || cuda_device >= ndev) return HB_ERR_CUDA;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, cuda_device) != cudaSuccess) return HB_ERR_CUDA;
    if (prop.major != 10 || prop.minor != 0) return HB_ERR_UNSUPPORTED;
    cudaGetDevice(&prev);
    if (cudaSetDevice(cuda_device) != cudaSuccess) return HB_ERR_CUDA;
    const int sms = prop.multiProcessorCount;
    void* scratch = nullptr;
    hb_status st = HB_OK;
    if (cudaMalloc(&scratch, 256) != cudaSuccess) st = HB_ERR_ALLOC;
    float ms = 0.f;
    const int blocks = sms * 8, iters = 1 << 14;
    const double chain_ops = (double)blocks * PK_THREADS * 8.0 * iters;
    if (st == HB_OK) {
        if (time_ms([&] { pk_ffma_kernel<<<blocks, PK_THREADS>>>((float*)scratch, iters, 0.999f, 0.001f); }, &ms) != cudaSuccess) st = HB_ERR_CUDA;
        else out5[0] = chain_ops / (ms * 1e-3) / 1e12;
    }
    if (st == HB_OK) {
        if (time_ms([&] { pk_dfma_kernel<<<blocks, PK_THREADS>>>((double*)scratch, iters / 4, 0.999, 0.001); }, &ms) != cudaSuccess) st = HB_ERR_CUDA;
        else out5[1] = chain_ops / 4.0 / (ms * 1e-3) / 1e12;
    }
    if (st == HB_OK) {
        if (time_ms([&] { pk_tanh_kernel<<<blocks, PK_THREADS>>>((float*)scratch, iters / 4); }, &ms) != cudaSuccess) st = HB_ERR_CUDA;
        else out5[2] = chain_ops / 4.0 / (ms * 1e-3) / 1e12;
    }
    const int reps = 4096;
    const size_t smem = 50 * 1024 + 1024;
    if (st == HB_OK) {
        cudaFuncSetAttribute(pk_mma_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (time_ms([&] { pk_mma_kernel<false><<<sms, 128, smem>>>(reps); }, &ms) != cudaSuccess) st = HB_ERR_CUDA;
        else out5[3] = (double)sms * reps * 4.0 * 2.0 * 128.0 * 256.0 * 16.0 / (ms * 1e-3) / 1e12;
    }
    if (st == HB_OK) {
        cudaFuncSetAttribute(pk_mma_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (time_ms([&] { pk_mma_kernel<true><<<sms, 128, smem>>>(reps); }, &ms) != cudaSuccess) st = HB_ERR_CUDA;
        else out5[4] = (double)sms * reps * 4.0 * 2.0 * 128.0 * 256.0 * 8.0 / (ms * 1e-3) / 1e12;
    }
    if (scratch) cudaFree(scratch);
    cudaSetDevice(prev);
    return st;
}
