// hb_internal.h -- shared declarations of libhb.so's translation units (host + device).
// Not part of the public ABI (include/hb.h) and not shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#define HB_MAX_LINEAR 12      // L_0 .. L_l, l <= 11 hidden layers
#define HB_MAX_WIDTH 1024
#define HB_NMOM 27            // 6 first + 21 second moments
#define HB_MOM_GRID_MAX 592    // 148 SMs x 4: most blocks one launch writes moment partials from
#define HB_MOM_MAX_BLOCKS 4736  // rows of a partials buffer: 8 launches (hb_push_host: one per chunk) x HB_MOM_GRID_MAX

// ---- conventional runs -------------------------------------------------------------------
struct HbRunMap {             // composed run: v' = M v (row-major 6x6, fp32, built in fp64 on the host)
    float m[36];
};

// pivot of the moment sums (a3): the nominal centroid of the state a monitor sees, tracked on the host through the
// lattice; the kernels accumulate sums of (v - pivot), the finalize adds it back to the means
struct HbPivot { double p[6]; };

// one conventional element in sequential mode (coefficients in fp64)
//  kind 0 drift : a0 = L, a1 = L/(bg)^2
//  kind 1 quad  : a0..a3 = x-plane 2x2 (row-major), a4..a7 = y-plane 2x2, a8 = L/(bg)^2
//  kind 2 sbend : a0..a3 = x-plane 2x2, a4 = R16, a5 = R26, a6 = L (y drift), a7 = R51, a8 = R52, a9 = R56
//  kind 3 exact drift (non-linear, R2x) : a0 = L, a1 = 1/beta0
//  kind 4 chromatic quad (non-linear, R3x) : a0 = L, a1 = k, a2 = 1/beta0
//  kind 5 thin multipole kick (non-linear for m > 2, R5x) : a0 = kn/(m-1)!, a1 = ks/(m-1)!, a2 = m
struct HbSeqElem {
    double a[10];
    int kind;
    int pad;
};

// ---- surrogate stage ---------------------------------------------------------------------
struct HbSurDev {             // passed by value to the surrogate kernels
    int n_linear;
    int act;                  // hb_act
    int coord;                // hb_coord
    int prec;                 // hb_prec
    int widths[HB_MAX_LINEAR + 1];
    float prelu[HB_MAX_LINEAR];
    // input normalisation  v^ = ((v - mu_hi) - mu_lo) * inv_sd   (mu split so that fp32 loses nothing)
    float mu_hi[6], mu_lo[6], inv_sd[6];
    // output  w = w^ * out_sd + out_mu
    float out_sd[6], out_mu[6];
    // COORD_T constants (R6, R7), all formed in fp64 on the host
    float bg0, g0;            // incoming reference
    float bg1, g1, inv_bg1;   // outgoing reference
    float uz_in_shift;        // (bg0 - in_mean[5])            : n5 = (duz + uz_in_shift) * inv_sd[5]
    float uz_out_shift;       // (out_mean[5] - bg1)           : d  = w^5 * out_sd[5] + uz_out_shift
    float z_out_mu;           // (out_mean[2] - z_ref)
    // fp32 path: packed W^T  [layer][k][npad]  and biases [layer][npad]
    const float* w32;
    const float* b32;
    long long w32_off[HB_MAX_LINEAR];
    int b32_off[HB_MAX_LINEAR];
    int npad32[HB_MAX_LINEAR];
    // tensor-core path: packed 16-bit (or tf32) operand image, see hb_sur_tc.cu
    const void* wtc;
    const float* btc;         // biases fp32, padded, per layer
    long long wtc_off[HB_MAX_LINEAR];   // byte offsets
    int btc_off[HB_MAX_LINEAR];
    int kpad[HB_MAX_LINEAR];  // padded fan-in  (multiple of 64 elements; layer 0: 64)
    int npadtc[HB_MAX_LINEAR];// padded fan-out (multiple of 16; hidden: multiple of 64)
    int tc_kind;              // which tensor-core kernel the image was packed for (hb_tc_choose, fixed at finalize)
    int tc_cg, tc_g, tc_occ;  // resident kernels: cluster size, epilogue warp groups, CTAs per SM (fixed at finalize)
    int fp32_tp;              // fp32 kernel: forced particles-per-block of the 4x4 shape, 0 = automatic (fixed at finalize)
    HbPivot mom_pivot;        // pivot of the fused moment sums of this stage's output (a3)
    unsigned char* act_scratch;   // wide nets (hb_sur_tcw.cu): two pre-tiled activation buffers of one chunk
};

struct HbParticles {
    float* v[6];              // x, px, y, py, t, pt
};

// ---- launchers (each returns the cudaError_t of the launch) ---------------------------------
// partials: device [>= gridDim][27] doubles or nullptr (no moments)
// pivot6_host: pivot of the fused moment sums (nullptr = zeros); unused without partials
cudaError_t hb_launch_run_composed(const HbParticles& p, size_t n, const HbRunMap& map, const double* pivot6_host,
                                   double* partials, int* nblocks_out, cudaStream_t s);
cudaError_t hb_launch_run_sequential(const HbParticles& p, size_t n, const HbSeqElem* d_elems, int count,
                                     bool fp32_regs, bool nonlinear, const double* pivot6_host, double* partials,
                                     int* nblocks_out, cudaStream_t s);
// sets the calling thread's hb_last_error() text (for entry points that live outside hb_api.cu)
void hb_internal_set_error(const char* msg);

cudaError_t hb_launch_moments_partials(const HbParticles& p, size_t n, const double* pivot6_host,
                                       double* partials, int* nblocks_out, cudaStream_t s);
// fixed-order sum of `nblocks` partials -> 27-double record (pivot added back to the means)
cudaError_t hb_launch_moments_finalize(const double* partials, int nblocks, size_t n,
                                       const double* pivot6_host, double* d_out27, cudaStream_t s);
// Surrogate launchers.  prepare = true (hb_lattice_finalize, once per stage): only set the launch attributes of the
// kernel instantiation the stage will use (dynamic shared memory), launch nothing.
// records of K linear images of a bunch from the bunch's record: d_rec_in 27 doubles, d_maps K x 36 (row-major), d_rec_out K x 27
cudaError_t hb_launch_candidates(const double* d_rec_in, const double* d_maps, int k_count, double* d_rec_out, cudaStream_t s);
cudaError_t hb_launch_sur_fp32(const HbParticles& p, size_t n, const HbSurDev& sd, double* partials,
                               int* nblocks_out, int sm_count, bool prepare, cudaStream_t s);
cudaError_t hb_launch_sur_tc(const HbParticles& p, size_t n, const HbSurDev& sd, double* partials,
                             int* nblocks_out, int sm_count, bool prepare, cudaStream_t s);
int hb_fp32_env_tp(void);     // HB_FP32_TP test hook (read at finalize)
// kernel and launch shape of a tensor-core stage (hb_sur_tc.cu; reads the test hooks of the environment): kind 0 = no
// schedule, 1 resident / one tile per CTA, 2 streamed, 3 layered, 4 resident / two tiles in flight
struct HbTcChoice { int kind, cg, g, occ; };
HbTcChoice hb_tc_choose(int prec, int n_linear, const int* widths);
// host-side packing for the tensor-core path (hb_sur_tc.cu owns the layout)
//  returns bytes needed; if dst != nullptr writes the image.  W row-major [out][in] fp32.
//  B: biases [out] fp32 per layer (the resident kernel's image carries those of the hidden layers; may be nullptr
//  when dst is).
size_t hb_tc_pack_weights(const HbTcChoice& ch, int prec, int n_linear, const int* widths, const float* const* W,
                          const float* const* B, void* dst, long long* off_bytes, int* kpad, int* npad);
bool hb_tc_supported(int prec, int n_linear, const int* widths, char* why, size_t why_len);
// streamed-weights variant (hb_sur_tcs.cu): hidden width <= 512, equal hidden widths, weights through an smem ring
bool hb_tcs_supported(int prec, int n_linear, const int* widths);   // prec: hb_prec (1 bf16, 2 f16, 3 tf32)
size_t hb_tcs_pack_weights(int prec, int n_linear, const int* widths, const float* const* W,
                           void* dst, long long* off_bytes, int* kpad, int* npad);
cudaError_t hb_launch_sur_tcs(const HbParticles& p, size_t n, const HbSurDev& sd, double* partials,
                              int* nblocks_out, int sm_count, bool prepare, cudaStream_t s);
// resident weights, two tiles in flight per CTA, hidden layers as N-halves (hb_sur_tc2.cu): hidden width 129..256
int hb_tc2_plan_cg(int n_linear, const int* widths, int force_cg);     // 0: no plan, else the cluster size
size_t hb_tc2_pack_weights(int prec, int cg, int n_linear, const int* widths, const float* const* W, const float* const* B,
                           void* dst, long long* off_bytes, int* kpad, int* npad);
cudaError_t hb_launch_sur_tc2(const HbParticles& p, size_t n, const HbSurDev& sd, double* partials,
                              int* nblocks_out, int sm_count, bool prepare, cudaStream_t s);
int hb_tc_kernel_kind(int prec, int n_linear, const int* widths);     // hb_tc_choose(...).kind
// wide nets (hidden width 513..1024, equal widths; bf16 / f16): hb_sur_tcw.cu
#define HB_TCW_CHUNK (1 << 20)        // particles per chunk (scratch: 2 buffers x chunk x padded width x 2 B)
bool hb_tcw_supported(int prec, int n_linear, const int* widths);
size_t hb_tcw_scratch_bytes(int n_linear, const int* widths);
size_t hb_tcw_pack_weights(int prec, int n_linear, const int* widths, const float* const* W,
                           void* dst, long long* off_bytes, int* kpad, int* npad);
cudaError_t hb_launch_sur_tcw(const HbParticles& p, size_t n, const HbSurDev& sd, double* partials, bool partials_zeroed,
                              int* nblocks_out, int sm_count, bool prepare, cudaStream_t s);
