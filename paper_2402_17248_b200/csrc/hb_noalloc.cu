// hb_noalloc.cu -- hb_moments_static(): the standalone moments pass (R10) for callers that cannot
// allocate device memory: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
//
// hb_moments() takes its block-partials scratch from the caller; here the scratch is a file-scope array in device
// memory.  Every GPU that loads libhb.so holds these HB_STATIC_SCRATCH_BYTES (27 x 4736 doubles = 999 KB) from the
// moment the module is loaded until the process exits.  The kernels are the ones hb_moments() launches
// (hb_moments_partials_kernel, hb_moments_finalize_kernel): same grid, same summation order, bit-identical records.
//
// In HOST code the name `hb_static_partials` is a host-side stand-in for the symbol, not a device address: a kernel
// given it would fault (or, where the GPU can reach host memory, use the wrong memory silently).  The device address
// is looked up once per device with cudaGetSymbolAddress(), with that device current, and that pointer is what the
// kernels receive.
//
// Sharing.  Every call on a device uses the same array.  A call's partials kernel overwrites the rows it will read
// (each of its blocks stores all 27 of its sums; nothing is accumulated into the array), so nothing has to start at
// zero and the contents left by the previous call are never read.  Two calls that OVERLAP on the GPU (different
// streams without an ordering between them) race on the array: order them on one stream or with events.
#include "../../include/hb.h"
#include "hb_internal.h"

#include <cstdint>
#include <cstdio>
#include <mutex>

namespace {

constexpr size_t HB_STATIC_SCRATCH_DOUBLES = (size_t)HB_NMOM * HB_MOM_MAX_BLOCKS;   // the layout hb_moments() uses
constexpr int HB_STATIC_MAX_DEVICES = 64;

static __device__ __align__(256) double hb_static_partials[HB_STATIC_SCRATCH_DOUBLES];

std::mutex g_mu;
double* g_dev_ptr[HB_STATIC_MAX_DEVICES];       // device address of hb_static_partials on device d (nullptr: not looked up)

hb_status na_fail(hb_status s, const char* msg) {
    hb_internal_set_error(msg);
    return s;
}

// the device address of the scratch on the CURRENT device (looked up on the first call for that device)
hb_status scratch_of_current_device(double** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return na_fail(HB_ERR_CUDA, cudaGetErrorString(e));
    if (dev < 0 || dev >= HB_STATIC_MAX_DEVICES) return na_fail(HB_ERR_UNSUPPORTED, "hb_moments_static: device ordinal above 63");
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_dev_ptr[dev]) {
        cudaDeviceProp prop;
        e = cudaGetDeviceProperties(&prop, dev);
        if (e != cudaSuccess) return na_fail(HB_ERR_CUDA, cudaGetErrorString(e));
        if (prop.major != 10 || prop.minor != 0)
            return na_fail(HB_ERR_UNSUPPORTED, "hb_moments_static: libhb is built for sm_100a (compute capability 10.0) only");
        double* ptr = nullptr;
        e = cudaGetSymbolAddress((void**)&ptr, hb_static_partials);
        if (e != cudaSuccess || !ptr) {
            char buf[256];
            snprintf(buf, sizeof buf, "hb_moments_static: cudaGetSymbolAddress(hb_static_partials) on device %d: %s", dev,
                     e != cudaSuccess ? cudaGetErrorString(e) : "null address");
            return na_fail(HB_ERR_CUDA, buf);
        }
        g_dev_ptr[dev] = ptr;
    }
    *out = g_dev_ptr[dev];
    return HB_OK;
}

}  // namespace

extern "C" size_t hb_moments_static_max_particles(void) { return (size_t)HB_MOMENTS_STATIC_MAX_N; }

extern "C" hb_status hb_moments_static(const float* x, const float* px, const float* y, const float* py, const float* t,
                                       const float* pt, size_t n, const double* pivot, double* d_out27, void* stream) {
    if (!d_out27) return na_fail(HB_ERR_INVALID_ARG, "hb_moments_static: d_out27 is NULL");
    if (n > (size_t)HB_MOMENTS_STATIC_MAX_N) {
        char buf[256];
        snprintf(buf, sizeof buf,
                 "hb_moments_static: n = %zu exceeds HB_MOMENTS_STATIC_MAX_N = %llu (the size this fixed-scratch entry point "
                 "is specified for); use hb_moments() with caller-owned scratch",
                 n, (unsigned long long)HB_MOMENTS_STATIC_MAX_N);
        return na_fail(HB_ERR_INVALID_ARG, buf);
    }
    cudaStream_t s = (cudaStream_t)stream;
    cudaError_t e;
    if (n == 0) {          // as hb_moments(): a record of NaNs
        e = cudaMemsetAsync(d_out27, 0xff, HB_NMOM * sizeof(double), s);
        return e == cudaSuccess ? HB_OK : na_fail(HB_ERR_CUDA, cudaGetErrorString(e));
    }
    const float* arr[6] = {x, px, y, py, t, pt};
    for (int j = 0; j < 6; ++j) {
        if (!arr[j]) return na_fail(HB_ERR_INVALID_ARG, "hb_moments_static: a particle array is NULL");
        if ((uintptr_t)arr[j] & 15u) return na_fail(HB_ERR_INVALID_ARG, "hb_moments_static: a particle array is not 16-byte aligned");
    }
    double* scratch = nullptr;
    const hb_status st = scratch_of_current_device(&scratch);
    if (st != HB_OK) return st;
    HbParticles p;
    for (int j = 0; j < 6; ++j) p.v[j] = const_cast<float*>(arr[j]);
    int nblocks = 0;
    e = hb_launch_moments_partials(p, n, pivot, scratch, &nblocks, s);
    if (e == cudaSuccess) e = hb_launch_moments_finalize(scratch, nblocks, n, pivot, d_out27, s);
    return e == cudaSuccess ? HB_OK : na_fail(HB_ERR_CUDA, cudaGetErrorString(e));
}
