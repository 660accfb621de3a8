// hb_device.cuh -- device helpers shared by libhb's kernels: moment accumulation (R10),
// s<->t conversion in deviation form (R6, R7), activations (Eq. 1, 2; tanh).
#pragma once
#include "hb_internal.h"

// ------------------------------------------------------------------------- moments (R10)
// Per-thread fp64 accumulators of the (pivot-shifted) raw sums:  S1_j = sum v_j,  S2_jk = sum v_j v_k (j<=k).
struct HbMomAcc {
    double s[HB_NMOM];
    __device__ __forceinline__ void clear() {
#pragma unroll
        for (int i = 0; i < HB_NMOM; ++i) s[i] = 0.0;
    }
    __device__ __forceinline__ void add(const double (&v)[6]) {
#pragma unroll
        for (int j = 0; j < 6; ++j) s[j] += v[j];
        int idx = 6;
#pragma unroll
        for (int j = 0; j < 6; ++j)
#pragma unroll
            for (int k = j; k < 6; ++k) { s[idx] = fma(v[j], v[k], s[idx]); ++idx; }
    }
    // one particle, shifted by the pivot (host-supplied nominal centroid: keeps E[v^2] - E[v]^2 well conditioned
    // for a bunch that sits far off axis with a small spread)
    __device__ __forceinline__ void add(const HbPivot& pv, float x, float px, float y, float py, float t, float pt) {
        const double v[6] = {(double)x - pv.p[0], (double)px - pv.p[1], (double)y - pv.p[2],
                             (double)py - pv.p[3], (double)t - pv.p[4], (double)pt - pv.p[5]};
        add(v);
    }
};

// Block-level fixed-order reduction of the 27 accumulators.  Inside a warp a reduce-scatter butterfly (step
// h = 16, 8, .., 1: each lane keeps one half of its values, sends the other half to lane ^ h and adds what it
// receives) leaves the warp total of moment l in lane l with 31 shuffles instead of 27 x 5; warp 0.. then sums the
// per-warp values in warp order.  `scratch`: shared, >= (blockDim/32)*27 doubles.  All threads of the
// participating group [tid0, tid0+nthreads) must call; `bar_id` named barrier.
// The block's 27 sums go to out_partial[j * HB_MOM_MAX_BLOCKS] (moment-major partials: the finalize kernel then
// reads every moment's row with consecutive lanes on consecutive addresses).
__device__ __forceinline__ void hb_block_reduce_moments(HbMomAcc& acc, double* scratch, double* out_partial,
                                                        int tid, int nthreads, int bar_id) {
    const int lane = tid & 31, warp = tid >> 5, nwarps = nthreads >> 5;
    double v[32];
#pragma unroll
    for (int i = 0; i < 32; ++i) v[i] = i < HB_NMOM ? acc.s[i] : 0.0;
#pragma unroll
    for (int h = 16; h >= 1; h >>= 1) {
        const bool upper = (lane & h) != 0;
#pragma unroll
        for (int i = 0; i < h; ++i) {
            if (i + h >= HB_NMOM && h == 16) {          // indices 27..31 are padding: nothing to send or keep
                const double send = upper ? v[i] : 0.0;
                const double got = __shfl_xor_sync(0xffffffffu, send, h);
                v[i] = upper ? 0.0 : v[i] + got;
            } else {
                const double keep = upper ? v[i + h] : v[i];
                const double send = upper ? v[i] : v[i + h];
                v[i] = keep + __shfl_xor_sync(0xffffffffu, send, h);
            }
        }
    }
    if (lane < HB_NMOM) scratch[warp * HB_NMOM + lane] = v[0];
    asm volatile("bar.sync %0, %1;" ::"r"(bar_id), "r"(nthreads) : "memory");
    if (tid < HB_NMOM) {
        double t = 0.0;
        for (int w = 0; w < nwarps; ++w) t += scratch[w * HB_NMOM + tid];
        out_partial[(size_t)tid * HB_MOM_MAX_BLOCKS] = t;
    }
}

// ------------------------------------------------------------------------- activations
__device__ __forceinline__ float hb_tanh_approx(float x) {
    float y;
    asm("tanh.approx.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

template <int ACT, bool FAST>
__device__ __forceinline__ float hb_activate(float z, float a) {
    if (ACT == 1) return fmaxf(z, 0.0f);                  // Eq. 1
    if (ACT == 2) return z >= 0.0f ? z : a * z;           // Eq. 2
    if (ACT == 3) return FAST ? hb_tanh_approx(z) : tanhf(z);
    return z;
}

// ------------------------------------------------------------------------- R6 / R8: prologue and epilogue
// s-coordinates of one particle -> the six NORMALISED network inputs.
__device__ __forceinline__ void hb_sur_prologue(const HbSurDev& sd, float x, float px, float y, float py,
                                                float t, float pt, float (&nin)[6]) {
    if (sd.coord == 0) {
        const float v[6] = {x, px, y, py, t, pt};
#pragma unroll
        for (int j = 0; j < 6; ++j) nin[j] = ((v[j] - sd.mu_hi[j]) - sd.mu_lo[j]) * sd.inv_sd[j];
    } else {
        // to_t in deviation form: never forms uz (~1958) and subtracts its mean in fp32
        const float ux = px * sd.bg0, uy = py * sd.bg0;
        const float dg = -pt * sd.bg0;                                   // gamma - gamma0
        const float g = sd.g0 + dg;
        const float num = fmaf(dg, 2.0f * sd.g0 + dg, -fmaf(ux, ux, uy * uy));  // uz^2 - uz0^2
        const float uz = sqrtf(fmaxf(fmaf(sd.bg0, sd.bg0, num), 0.0f));
        const float duz = num / (uz + sd.bg0);                           // uz - uz0
        const float ig = 1.0f / g;
        const float xt = fmaf(-ux * ig, t, x);
        const float yt = fmaf(-uy * ig, t, y);
        const float zt = -(uz * ig) * t;
        const float v[5] = {xt, yt, zt, ux, uy};
#pragma unroll
        for (int j = 0; j < 5; ++j) nin[j] = ((v[j] - sd.mu_hi[j]) - sd.mu_lo[j]) * sd.inv_sd[j];
        nin[5] = (duz + sd.uz_in_shift) * sd.inv_sd[5];
    }
}

// six raw network outputs -> s-coordinates (about the new reference for COORD_T)
__device__ __forceinline__ void hb_sur_epilogue(const HbSurDev& sd, const float (&w)[6], float& x, float& px,
                                                float& y, float& py, float& t, float& pt) {
    if (sd.coord == 0) {
        x = fmaf(w[0], sd.out_sd[0], sd.out_mu[0]);
        px = fmaf(w[1], sd.out_sd[1], sd.out_mu[1]);
        y = fmaf(w[2], sd.out_sd[2], sd.out_mu[2]);
        py = fmaf(w[3], sd.out_sd[3], sd.out_mu[3]);
        t = fmaf(w[4], sd.out_sd[4], sd.out_mu[4]);
        pt = fmaf(w[5], sd.out_sd[5], sd.out_mu[5]);
    } else {
        const float xt = fmaf(w[0], sd.out_sd[0], sd.out_mu[0]);
        const float yt = fmaf(w[1], sd.out_sd[1], sd.out_mu[1]);
        const float zt = fmaf(w[2], sd.out_sd[2], sd.z_out_mu);          // z - z_ref  (R7)
        const float ux = fmaf(w[3], sd.out_sd[3], sd.out_mu[3]);
        const float uy = fmaf(w[4], sd.out_sd[4], sd.out_mu[4]);
        const float d = fmaf(w[5], sd.out_sd[5], sd.uz_out_shift);       // uz - uz1
        const float uz = sd.bg1 + d;
        const float s2 = fmaf(ux, ux, uy * uy);
        const float g = sqrtf(1.0f + s2 + uz * uz);
        const float dgam = fmaf(d, 2.0f * sd.bg1 + d, s2) / (g + sd.g1); // gamma - gamma1
        const float iuz = 1.0f / uz;
        x = fmaf(-ux * iuz, zt, xt);
        y = fmaf(-uy * iuz, zt, yt);
        t = -zt * g * iuz;
        px = ux * sd.inv_bg1;
        py = uy * sd.inv_bg1;
        pt = -dgam * sd.inv_bg1;
    }
}
