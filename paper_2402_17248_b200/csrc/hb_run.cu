// hb_run.cu -- fused conventional-run kernels (a2), moment partials / finalize (a3).
//
// Row a2 of the hot path: a whole run of consecutive conventional elements (drift R2,
// thick quad R3, sector bend R4) is applied with ONE read and ONE write of the six
// SoA arrays: 48 B per particle per run, HBM-bound.  Loads/stores are 128-bit (4 particles per
// thread per coordinate), streaming (evict-first) cache hints, in place.
//   composed  : v' = M_run v, M_run concatenated in fp64 on the host, 36 FFMA per particle.
//   sequential: element list staged in shared memory, applied one by one in registers
//               (fp64, or fp32 for HB_RUN_SEQUENTIAL_FP32), one rounding at the store.
// Row a3: when a monitor follows the run, the 27 raw moment sums (R10) are accumulated in fp64 from
// the values already in registers, reduced by warp shuffles, and one partial per block is written.
#include "hb_device.cuh"

#define RUN_THREADS 256

__device__ __forceinline__ float4 ld_stream(const float* p) { return __ldcs(reinterpret_cast<const float4*>(p)); }
__device__ __forceinline__ void st_stream(float* p, const float4& v) { __stcs(reinterpret_cast<float4*>(p), v); }

__device__ __forceinline__ void apply_map(const HbRunMap& M, const float (&in)[6], float (&out)[6]) {
#pragma unroll
    for (int r = 0; r < 6; ++r) {
        float acc = M.m[r * 6] * in[0];
#pragma unroll
        for (int c = 1; c < 6; ++c) acc = fmaf(M.m[r * 6 + c], in[c], acc);
        out[r] = acc;
    }
}

template <bool MOM>
__global__ void __launch_bounds__(RUN_THREADS, MOM ? 2 : 4)
hb_run_composed_kernel(HbParticles p, size_t n, const __grid_constant__ HbRunMap M, const __grid_constant__ HbPivot pv,
                       double* __restrict__ partials) {
    __shared__ double red[(RUN_THREADS / 32) * HB_NMOM];
    HbMomAcc acc;
    if (MOM) acc.clear();
    const size_t nq = n >> 2;
    const size_t stride = (size_t)gridDim.x * RUN_THREADS;
    for (size_t q = (size_t)blockIdx.x * RUN_THREADS + threadIdx.x; q < nq; q += stride) {
        float4 c[6];
#pragma unroll
        for (int j = 0; j < 6; ++j) c[j] = ld_stream(p.v[j] + 4 * q);
        float4 o[6];
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            float in[6], out[6];
#pragma unroll
            for (int j = 0; j < 6; ++j) in[j] = reinterpret_cast<const float*>(&c[j])[e];
            apply_map(M, in, out);
#pragma unroll
            for (int j = 0; j < 6; ++j) reinterpret_cast<float*>(&o[j])[e] = out[j];
            if (MOM) acc.add(pv, out[0], out[1], out[2], out[3], out[4], out[5]);
        }
#pragma unroll
        for (int j = 0; j < 6; ++j) st_stream(p.v[j] + 4 * q, o[j]);
    }
    // ragged tail (n mod 4 particles): scalar, by the first threads of block 0
    if (blockIdx.x == 0 && threadIdx.x < (n & 3)) {
        const size_t i = (nq << 2) + threadIdx.x;
        float in[6], out[6];
#pragma unroll
        for (int j = 0; j < 6; ++j) in[j] = p.v[j][i];
        apply_map(M, in, out);
#pragma unroll
        for (int j = 0; j < 6; ++j) p.v[j][i] = out[j];
        if (MOM) acc.add(pv, out[0], out[1], out[2], out[3], out[4], out[5]);
    }
    if (MOM) hb_block_reduce_moments(acc, red, partials + blockIdx.x, threadIdx.x, RUN_THREADS, 1);
}

// ---------------------------------------------------------------------------------- sequential
#define SEQ_CHUNK 128
template <typename T>
struct SeqElemT { T a[10]; int kind; };

// NL: the run holds non-linear elements (kinds 3-5); the linear-only instantiation keeps the lean three-way branch
template <typename T, bool NL>
__device__ __forceinline__ void seq_apply(const SeqElemT<T>& e, T (&v)[6]) {
    // v = (x, px, y, py, t, pt); pt never changes (R2-R5x)
    if (e.kind == 0) {                 // drift R2
        v[0] = fma(e.a[0], v[1], v[0]);
        v[2] = fma(e.a[0], v[3], v[2]);
        v[4] = fma(e.a[1], v[5], v[4]);
    } else if (e.kind == 1) {          // thick quad R3
        const T x = v[0], px = v[1], y = v[2], py = v[3];
        v[0] = fma(e.a[0], x, e.a[1] * px);
        v[1] = fma(e.a[2], x, e.a[3] * px);
        v[2] = fma(e.a[4], y, e.a[5] * py);
        v[3] = fma(e.a[6], y, e.a[7] * py);
        v[4] = fma(e.a[8], v[5], v[4]);
    } else if (NL && e.kind == 3) {    // exact drift R2x (non-linear): a0 = L, a1 = 1/beta0
        // pz^2 = (1/beta0 - pt)^2 - 1/(beta0 gamma0)^2 - px^2 - py^2 = 1 - 2 pt/beta0 + pt^2 - px^2 - py^2
        const T px = v[1], py = v[3], pt = v[5];
        const T pz2 = fma(pt, pt - T(2) * e.a[1], T(1)) - fma(px, px, py * py);
        const T ipz = T(1) / sqrt(pz2);
        v[0] = fma(e.a[0] * ipz, px, v[0]);
        v[2] = fma(e.a[0] * ipz, py, v[2]);
        v[4] = fma(e.a[0], fma(e.a[1] - pt, ipz, -e.a[1]), v[4]);
    } else if (NL && e.kind == 4) {    // chromatic thick quad R3x (non-linear): a0 = L, a1 = k, a2 = 1/beta0
        const T L = e.a[0], k = e.a[1], pt = v[5];
        const T en = e.a[2] - pt;                                   // E / (p0 c)
        const T d1 = sqrt(fma(pt, pt - T(2) * e.a[2], T(1)));       // 1 + delta = |p| / p0
        T I = T(0);                                                 // integral of px^2 + py^2 over the element
#pragma unroll
        for (int pl = 0; pl < 2; ++pl) {
            const T kp = pl == 0 ? k : -k;
            const T u0 = v[2 * pl], p0 = v[2 * pl + 1];
            if (kp > T(0)) {
                const T w = sqrt(kp / d1), c = cos(w * L), sn = sin(w * L), B = -w * d1 * u0;
                v[2 * pl] = fma(c, u0, sn / (w * d1) * p0);
                v[2 * pl + 1] = fma(B, sn, p0 * c);
                I += T(0.5) * (p0 * p0 + B * B) * L + (p0 * p0 - B * B) * sin(T(2) * w * L) / (T(4) * w) +
                     p0 * B * (T(1) - cos(T(2) * w * L)) / (T(2) * w);
            } else if (kp < T(0)) {
                const T w = sqrt(-kp / d1), c = cosh(w * L), sn = sinh(w * L), B = w * d1 * u0;
                v[2 * pl] = fma(c, u0, sn / (w * d1) * p0);
                v[2 * pl + 1] = fma(B, sn, p0 * c);
                I += T(0.5) * (p0 * p0 - B * B) * L + (p0 * p0 + B * B) * sinh(T(2) * w * L) / (T(4) * w) +
                     p0 * B * (cosh(T(2) * w * L) - T(1)) / (T(2) * w);
            } else {
                v[2 * pl] = fma(L / d1, p0, u0);
                I += p0 * p0 * L;
            }
        }
        v[4] += L * (en / d1 - e.a[2]) + en * I / (T(2) * d1 * d1 * d1);
    } else if (NL && e.kind == 5) {    // thin multipole kick R5x: a0 = kn/(m-1)!, a1 = ks/(m-1)!, a2 = m
        const int m = (int)e.a[2];
        T zr = T(1), zi = T(0);
        for (int j = 1; j < m; ++j) {
            const T r = zr * v[0] - zi * v[2], im = zr * v[2] + zi * v[0];
            zr = r; zi = im;
        }
        v[1] -= e.a[0] * zr - e.a[1] * zi;
        v[3] += e.a[0] * zi + e.a[1] * zr;
    } else {                           // sector bend R4
        const T x = v[0], px = v[1], d = v[5];
        v[0] = fma(e.a[0], x, fma(e.a[1], px, e.a[4] * d));
        v[1] = fma(e.a[2], x, fma(e.a[3], px, e.a[5] * d));
        v[2] = fma(e.a[6], v[3], v[2]);
        v[4] = fma(e.a[7], x, fma(e.a[8], px, fma(e.a[9], d, v[4])));
    }
}

// Three blocks per SM (80 registers) for the linear elements: the kernel waits on dependent DFMAs (ncu: 35 % of the stall
// samples are fixed-latency waits at 16 warps per SM), 2.47 -> 2.19 ms on C2; the non-linear elements (square roots and
// divisions in fp64) spill at 80 registers and stay at two blocks.
template <typename T, bool MOM, bool NL>
__global__ void __launch_bounds__(RUN_THREADS, NL ? 2 : 3)
hb_run_sequential_kernel(HbParticles p, size_t n, const HbSeqElem* __restrict__ elems, int count,
                         const __grid_constant__ HbPivot pv, double* __restrict__ partials) {
    __shared__ SeqElemT<T> se[SEQ_CHUNK];
    __shared__ double red[(RUN_THREADS / 32) * HB_NMOM];
    HbMomAcc acc;
    if (MOM) acc.clear();
    const size_t nq = n >> 2;
    const size_t nwork = nq + ((n & 3) ? 1 : 0);           // last work item = ragged tail
    const size_t stride = (size_t)gridDim.x * RUN_THREADS;
    const size_t first = (size_t)blockIdx.x * RUN_THREADS + threadIdx.x;
    // every thread of the block runs the same number of outer iterations (the element staging syncs)
    const size_t base0 = (size_t)blockIdx.x * RUN_THREADS;
    for (size_t base = base0; base < nwork; base += stride) {
        const size_t q = base + threadIdx.x;
        const bool active = q < nwork;
        const bool tail = active && q == nq;
        const int cnt = !active ? 0 : (tail ? (int)(n & 3) : 4);
        T v[4][6];
        if (active && !tail) {
            float4 c[6];
#pragma unroll
            for (int j = 0; j < 6; ++j) c[j] = ld_stream(p.v[j] + 4 * q);
#pragma unroll
            for (int e = 0; e < 4; ++e)
#pragma unroll
                for (int j = 0; j < 6; ++j) v[e][j] = (T) reinterpret_cast<const float*>(&c[j])[e];
        } else {
#pragma unroll
            for (int e = 0; e < 4; ++e)
#pragma unroll
                for (int j = 0; j < 6; ++j) v[e][j] = (e < cnt) ? (T)p.v[j][4 * nq + e] : (T)0;
        }
        for (int c0 = 0; c0 < count; c0 += SEQ_CHUNK) {
            const int m = min(SEQ_CHUNK, count - c0);
            __syncthreads();
            for (int i = threadIdx.x; i < m; i += RUN_THREADS) {
                const HbSeqElem& g = elems[c0 + i];
#pragma unroll
                for (int k = 0; k < 10; ++k) se[i].a[k] = (T)g.a[k];
                se[i].kind = g.kind;
            }
            __syncthreads();
            for (int i = 0; i < m; ++i) {
                const SeqElemT<T> e = se[i];
#pragma unroll
                for (int k = 0; k < 4; ++k) seq_apply<T, NL>(e, v[k]);
            }
        }
        if (active && !tail) {
            float4 o[6];
#pragma unroll
            for (int e = 0; e < 4; ++e)
#pragma unroll
                for (int j = 0; j < 6; ++j) reinterpret_cast<float*>(&o[j])[e] = (float)v[e][j];
#pragma unroll
            for (int j = 0; j < 6; ++j) st_stream(p.v[j] + 4 * q, o[j]);
        } else {
#pragma unroll
            for (int e = 0; e < 4; ++e)
                if (e < cnt)
#pragma unroll
                    for (int j = 0; j < 6; ++j) p.v[j][4 * nq + e] = (float)v[e][j];
        }
        if (MOM) {
#pragma unroll
            for (int e = 0; e < 4; ++e)
                if (e < cnt)
                    acc.add(pv, (float)v[e][0], (float)v[e][1], (float)v[e][2], (float)v[e][3], (float)v[e][4],
                            (float)v[e][5]);
        }
    }
    (void)first;
    if (MOM) hb_block_reduce_moments(acc, red, partials + blockIdx.x, threadIdx.x, RUN_THREADS, 1);
}

// ---------------------------------------------------------------------------------- standalone moments
__global__ void __launch_bounds__(RUN_THREADS, 2)
hb_moments_partials_kernel(HbParticles p, size_t n, const __grid_constant__ HbPivot pv, double* __restrict__ partials) {
    __shared__ double red[(RUN_THREADS / 32) * HB_NMOM];
    HbMomAcc acc;
    acc.clear();
    const size_t nq = n >> 2;
    const size_t stride = (size_t)gridDim.x * RUN_THREADS;
    for (size_t q = (size_t)blockIdx.x * RUN_THREADS + threadIdx.x; q < nq; q += stride) {
        float4 c[6];
#pragma unroll
        for (int j = 0; j < 6; ++j) c[j] = ld_stream(p.v[j] + 4 * q);
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            double v[6];
#pragma unroll
            for (int j = 0; j < 6; ++j) v[j] = (double)reinterpret_cast<const float*>(&c[j])[e] - pv.p[j];
            acc.add(v);
        }
    }
    if (blockIdx.x == 0 && threadIdx.x < (n & 3)) {
        const size_t i = (nq << 2) + threadIdx.x;
        double v[6];
#pragma unroll
        for (int j = 0; j < 6; ++j) v[j] = (double)p.v[j][i] - pv.p[j];
        acc.add(v);
    }
    hb_block_reduce_moments(acc, red, partials + blockIdx.x, threadIdx.x, RUN_THREADS, 1);
}

// One block of 27 warps: warp j sums partial[j][k] (moment-major), k = lane, lane+32, ... in a fixed order (loads issued eight
// at a time so that their latencies overlap), then an xor-shuffle tree.  Threads 0..26 turn the raw sums into the
// record (means + centred covariance, 1/N).
#define FIN_THREADS (HB_NMOM * 32)
__global__ void __launch_bounds__(FIN_THREADS, 1)
hb_moments_finalize_kernel(const double* __restrict__ partials, int nblocks, size_t n,
                           const __grid_constant__ HbPivot pv, double* __restrict__ out) {
    __shared__ double S[HB_NMOM];
    const int j = threadIdx.x >> 5, lane = threadIdx.x & 31;
    // launched with programmatic stream serialization: the block may become resident while the producing kernel is
    // still draining; its partials are complete and visible once this returns
    asm volatile("griddepcontrol.wait;" ::: "memory");
    double v = 0.0;
    // FIN_BATCH loads in flight per lane: one launch's partials (<= 592 blocks) are one batch; same summation order
    // as a plain ascending loop over this lane's blocks
    constexpr int FIN_BATCH = 20;
    for (int k0 = lane; k0 < nblocks; k0 += 32 * FIN_BATCH) {
        double t[FIN_BATCH];
#pragma unroll
        for (int u = 0; u < FIN_BATCH; ++u) {
            const int k = k0 + 32 * u;
            t[u] = k < nblocks ? __ldcg(partials + (size_t)j * HB_MOM_MAX_BLOCKS + k) : 0.0;
        }
#pragma unroll
        for (int u = 0; u < FIN_BATCH; ++u) v += t[u];
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if (lane == 0) S[j] = v;
    __syncthreads();
    if (threadIdx.x < HB_NMOM) {
        const int i = threadIdx.x;
        const double inv = n > 0 ? 1.0 / (double)n : __longlong_as_double(0x7ff8000000000000LL);
        if (i < 6) {
            out[i] = S[i] * inv + pv.p[i];
        } else {
            int a = 0, rem = i - 6;
            while (rem >= 6 - a) { rem -= 6 - a; ++a; }
            const int b = a + rem;
            out[i] = S[i] * inv - (S[a] * inv) * (S[b] * inv);
        }
    }
}

// ---------------------------------------------------------------------------------- launchers
static HbPivot make_pivot(const double* pivot6_host) {
    HbPivot pv;
    for (int j = 0; j < 6; ++j) pv.p[j] = pivot6_host ? pivot6_host[j] : 0.0;
    return pv;
}

static int run_grid(size_t n, bool moments) {
    const size_t nq = (n >> 2) + ((n & 3) ? 1 : 0);
    size_t blocks = (nq + RUN_THREADS - 1) / RUN_THREADS;
    if (blocks < 1) blocks = 1;
    const size_t cap = moments ? HB_MOM_GRID_MAX : 148 * 32;   // moments: 592 = 148 x 4 (2 resident x 2 waves)
    if (blocks > cap) blocks = cap;
    return (int)blocks;
}

cudaError_t hb_launch_run_composed(const HbParticles& p, size_t n, const HbRunMap& map, const double* pivot6_host,
                                   double* partials, int* nblocks_out, cudaStream_t s) {
    const int grid = run_grid(n, partials != nullptr);
    if (nblocks_out) *nblocks_out = grid;
    const HbPivot pv = make_pivot(pivot6_host);
    if (partials)
        hb_run_composed_kernel<true><<<grid, RUN_THREADS, 0, s>>>(p, n, map, pv, partials);
    else
        hb_run_composed_kernel<false><<<grid, RUN_THREADS, 0, s>>>(p, n, map, pv, partials);
    return cudaGetLastError();
}

cudaError_t hb_launch_run_sequential(const HbParticles& p, size_t n, const HbSeqElem* d_elems, int count,
                                     bool fp32_regs, bool nonlinear, const double* pivot6_host, double* partials,
                                     int* nblocks_out, cudaStream_t s) {
    const int grid = run_grid(n, partials != nullptr);
    if (nblocks_out) *nblocks_out = grid;
    const HbPivot pv = make_pivot(pivot6_host);
    if (nonlinear) {          // non-linear elements: fp64 registers only
        if (partials) hb_run_sequential_kernel<double, true, true><<<grid, RUN_THREADS, 0, s>>>(p, n, d_elems, count, pv, partials);
        else hb_run_sequential_kernel<double, false, true><<<grid, RUN_THREADS, 0, s>>>(p, n, d_elems, count, pv, partials);
    } else if (fp32_regs) {
        if (partials) hb_run_sequential_kernel<float, true, false><<<grid, RUN_THREADS, 0, s>>>(p, n, d_elems, count, pv, partials);
        else hb_run_sequential_kernel<float, false, false><<<grid, RUN_THREADS, 0, s>>>(p, n, d_elems, count, pv, partials);
    } else {
        if (partials) hb_run_sequential_kernel<double, true, false><<<grid, RUN_THREADS, 0, s>>>(p, n, d_elems, count, pv, partials);
        else hb_run_sequential_kernel<double, false, false><<<grid, RUN_THREADS, 0, s>>>(p, n, d_elems, count, pv, partials);
    }
    return cudaGetLastError();
}

cudaError_t hb_launch_moments_partials(const HbParticles& p, size_t n, const double* pivot6_host, double* partials,
                                       int* nblocks_out, cudaStream_t s) {
    const HbPivot pv = make_pivot(pivot6_host);
    const int grid = run_grid(n, true);
    if (nblocks_out) *nblocks_out = grid;
    hb_moments_partials_kernel<<<grid, RUN_THREADS, 0, s>>>(p, n, pv, partials);
    return cudaGetLastError();
}

cudaError_t hb_launch_moments_finalize(const double* partials, int nblocks, size_t n, const double* pivot6_host,
                                       double* d_out27, cudaStream_t s) {
    const HbPivot pv = make_pivot(pivot6_host);
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(1);
    cfg.blockDim = dim3(FIN_THREADS);
    cfg.dynamicSmemBytes = 0;
    cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    cudaError_t e = cudaLaunchKernelEx(&cfg, hb_moments_finalize_kernel, partials, nblocks, n, pv, d_out27);
    return e != cudaSuccess ? e : cudaGetLastError();
}

// ---------------------------------------------------------------------------------- candidate maps (NEXT-4)
// Records of the images  M_k v  of one bunch under K linear maps, from the bunch's own record: for a linear map the mean
// and the centred second moments transform exactly,  m' = M m,  C' = M C M^T  (sample moments, not a statistical statement),
// so K candidate settings of a transport section cost ONE pass over the particles (24 B each, hb_moments_partials_kernel)
// whatever K is.  One thread per candidate: 6 x 6 products in fp64.
__global__ void hb_candidates_kernel(const double* __restrict__ rec_in, const double* __restrict__ maps, int k_count,
                                     double* __restrict__ rec_out) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= k_count) return;
    const double* M = maps + (size_t)k * 36;
    double m[6], C[6][6];
    for (int i = 0; i < 6; ++i) m[i] = rec_in[i];
    int idx = 6;
    for (int i = 0; i < 6; ++i)
        for (int j = i; j < 6; ++j) { C[i][j] = rec_in[idx]; C[j][i] = rec_in[idx]; ++idx; }
    double* out = rec_out + (size_t)k * HB_NMOM;
    for (int i = 0; i < 6; ++i) {
        double a = 0.0;
        for (int j = 0; j < 6; ++j) a = fma(M[i * 6 + j], m[j], a);
        out[i] = a;
    }
    double T[6][6];                        // T = M C
    for (int i = 0; i < 6; ++i)
        for (int j = 0; j < 6; ++j) {
            double a = 0.0;
            for (int q = 0; q < 6; ++q) a = fma(M[i * 6 + q], C[q][j], a);
            T[i][j] = a;
        }
    idx = 6;
    for (int i = 0; i < 6; ++i)
        for (int j = i; j < 6; ++j) {
            double a = 0.0;
            for (int q = 0; q < 6; ++q) a = fma(T[i][q], M[j * 6 + q], a);
            out[idx++] = a;
        }
}

cudaError_t hb_launch_candidates(const double* d_rec_in, const double* d_maps, int k_count, double* d_rec_out, cudaStream_t s) {
    if (k_count <= 0) return cudaSuccess;
    hb_candidates_kernel<<<(k_count + 63) / 64, 64, 0, s>>>(d_rec_in, d_maps, k_count, d_rec_out);
    return cudaGetLastError();
}
