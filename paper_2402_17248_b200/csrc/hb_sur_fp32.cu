// hb_sur_fp32.cu -- surrogate stage on the CUDA cores (HB_PREC_FP32): rows a4-a6 with an FFMA GEMM chain.
//
// One block owns a tile of TP particles.  Activations live in shared memory as [feature][particle]
// (two ping-pong buffers); the transposed weights W^T [k][n] (packed, zero-padded to 64 outputs, by
// hb_api.cu) are streamed through two [KCH][OCB] shared slabs filled by cp.async (slab c + 1 lands while
// slab c is multiplied: one barrier per slab).  Each thread owns a 4 x 4 or 8 x 8 (particles x outputs) register
// tile; the operands of k step k + 1 are loaded before the FFMAs of step k.  The kernel is bound by the shared-memory
// data path, so the lane -> (particle group, output group) map is the one for which ncu counts two wavefronts
// per LDS.128 for both operands (profiles/r1_fp32.md).  Partial sums of each 32-wide K span are formed
// separately and then added (shorter rounding chains), bias is added last in fp32, tanh is tanhf.
// Prologue (s->t R6, normalise R8) and epilogue (de-normalise R8, reference R7, t->s R6, moments R10)
// are fused: hidden activations never touch HBM (data preparation is 1-2 % of the push).
#include "hb_device.cuh"

#include <cstdlib>

#define KC 16
#define OC 64

// Two fp32 FMAs per instruction (sm_100: fma.rn.f32x2, SASS FFMA2): d.lo = a.lo * b.lo + c.lo, d.hi likewise, each rounded
// exactly as a scalar fmaf.  The register tile's outer product issues (4R)^2 / 2 of these per k step instead of (4R)^2
// FFMA; ptxas folds the duplicated activation of pk2(a, a) into the instruction's scalar-broadcast operand (no moves).
// Why: the scalar kernel was bound by instruction issue and operand dispatch, not by the FMA pipe (ncu: issue slots
// 72.9 % busy, 0.34 dispatch-stall cycles per issued instruction, FMA pipe 63 %).
__device__ __forceinline__ unsigned long long pk2(float lo, float hi) {
    unsigned long long d;
    asm("mov.b64 %0, {%1, %2};" : "=l"(d) : "f"(lo), "f"(hi));
    return d;
}
__device__ __forceinline__ void unpk2(unsigned long long v, float& lo, float& hi) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ unsigned long long fma2(unsigned long long a, unsigned long long b, unsigned long long c) {
    unsigned long long d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ unsigned long long add2(unsigned long long a, unsigned long long b) {
    unsigned long long d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}

// R = 1: 4 x 4 register tile, OCB = 64-wide output blocks; R = 2: 8 x 8 register tile (two float4 per operand and
// k step: half the shared-memory wavefronts per FFMA) with OCB = 256 (one 256-thread block of 64 particles per SM, two
// warps per scheduler at ~240 registers) or OCB = 128 (two 128-thread blocks per SM).  KCH = rows per weight slab.
template <int TP, int ACT, bool MOM, int R, int OCB, int KCH>
__global__ void __launch_bounds__((TP / (4 * R)) * (OCB / (4 * R)), R == 2 ? (OCB == 128 ? 2 : 1) : (TP == 64 ? 1 : 3))
hb_sur_fp32_kernel(HbParticles p, size_t n, const __grid_constant__ HbSurDev sd, int hmax, double* __restrict__ partials) {
    constexpr int NT = (TP / (4 * R)) * (OCB / (4 * R));
    extern __shared__ __align__(16) float smem[];
    float* actA = smem;                          // [hmax][TP]
    float* actB = actA + (size_t)hmax * TP;      // [hmax][TP]
    float* Ws = actB + (size_t)hmax * TP;        // [2][KCH][OCB]
    double* red = reinterpret_cast<double*>(Ws + 2 * KCH * OCB);
    const uint32_t ws_addr = (uint32_t)__cvta_generic_to_shared(Ws);

    const int tid = threadIdx.x;
    // Activation rows are XOR-swizzled: the 16-byte chunk (4 particles) q of feature row f sits at chunk q ^ SWZ(f),
    // SWZ(f) = ((f >> 2) & 3) << 1.  A k step reads ONE row (every lane the same f: a permutation, still two wavefronts
    // per LDS.128); the store of a finished output block writes FOUR rows per quarter warp (rows 4 apart, the same
    // chunks): unswizzled that was 16 wavefronts per STS.128 (ncu: 13.2-way store conflicts, 11 % of all shared-memory
    // wavefronts), swizzled it is 4, the minimum for 512 bytes.
    constexpr int SWM = TP >= 32 ? 3 : 0;
    auto act_idx = [&](int f, int e) -> size_t {
        return (size_t)f * TP + (size_t)(((((e >> 2) ^ (((f >> 2) & SWM) << 1)) << 2) | (e & 3)));
    };
    // a warp = 8 particle groups x 4 output groups.  Lane bits (4,3,0) pick the particle group and bits (2,1) the
    // output group: both LDS.128 of a k step then cost two shared-memory wavefronts (with output group = lane % 4
    // the weight load took four: ncu, L1 Wavefronts Shared per instruction)
    constexpr int P = TP / (4 * R), PW = P >= 8 ? 8 : P, OW = 32 / PW;     // particle / output groups per warp
    const int lane = tid & 31;
    const int ol = PW == 8 ? ((lane >> 1) & 3) : lane % OW;
    const int pl = PW == 8 ? ((lane & 1) | ((lane >> 3) << 1)) : lane / OW;
    const int og = ((tid >> 5) / (P / PW)) * OW + ol;
    const int pg = ((tid >> 5) % (P / PW)) * PW + pl;
    // float offset of this thread's particle chunk in a row of swizzle class c (compile-time c: a register per class)
    auto pgx = [&](int c) -> int { return 4 * (pg ^ ((c & SWM) << 1)); };
    const int pgx_out = pgx(og);                 // ... in the rows this thread stores (class og & 3)
    HbMomAcc acc;
    if (MOM) acc.clear();
    int c = 0;                                   // running K-chunk counter (selects the weight-slab buffer)
    const size_t ntiles = (n + TP - 1) / TP;

    for (size_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const size_t i0 = tile * TP;
        __syncthreads();
        if (tid < TP) {
            const size_t i = i0 + tid;
            float nin[6] = {0, 0, 0, 0, 0, 0};
            if (i < n) hb_sur_prologue(sd, p.v[0][i], p.v[1][i], p.v[2][i], p.v[3][i], p.v[4][i], p.v[5][i], nin);
#pragma unroll
            for (int j = 0; j < 6; ++j) actA[act_idx(j, tid)] = nin[j];
        }
        float* in = actA;
        float* out = actB;
        for (int l = 0; l < sd.n_linear; ++l) {
            const int K = sd.widths[l], npad = sd.npad32[l];
            const float* __restrict__ Wt = sd.w32 + sd.w32_off[l];
            const float* __restrict__ bias = sd.b32 + sd.b32_off[l];
            const bool last = (l == sd.n_linear - 1);
            const float slope = sd.prelu[l];
            if (last && sd.widths[l + 1] <= 8) {
                // Narrow output layer (6 of the 64 padded outputs are real): thread = (particle, quarter of K),
                // six dot products over its K quarter, partial sums through the free activation buffer.  The
                // weight row is the same address for a whole warp (one broadcast load from L1).
                constexpr int NQ = NT / TP;                      // = 4
                const int nout = sd.widths[l + 1];
                const int pl_ = tid % TP, kq = tid / TP;
                const int KQ = (K + NQ - 1) / NQ;
                const int kb = kq * KQ, ke = min(K, kb + KQ);
                float d[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
                __syncthreads();                                 // layer input complete
#pragma unroll 4
                for (int k = kb; k < ke; ++k) {
                    const float a = in[act_idx(k, pl_)];
                    const float4 w0 = __ldg(reinterpret_cast<const float4*>(Wt + (size_t)k * npad));
                    const float4 w1 = __ldg(reinterpret_cast<const float4*>(Wt + (size_t)k * npad) + 1);
                    d[0] = fmaf(a, w0.x, d[0]); d[1] = fmaf(a, w0.y, d[1]);
                    d[2] = fmaf(a, w0.z, d[2]); d[3] = fmaf(a, w0.w, d[3]);
                    d[4] = fmaf(a, w1.x, d[4]); d[5] = fmaf(a, w1.y, d[5]);
                    d[6] = fmaf(a, w1.z, d[6]); d[7] = fmaf(a, w1.w, d[7]);
                }
#pragma unroll
                for (int j = 0; j < 8; ++j) out[(size_t)(8 + j * NQ + kq) * TP + pl_] = d[j];
                __syncthreads();
                if (tid < TP) {
#pragma unroll
                    for (int j = 0; j < 8; ++j) {
                        float z = 0.0f;
#pragma unroll
                        for (int q = 0; q < NQ; ++q) z += out[(size_t)(8 + j * NQ + q) * TP + tid];
                        if (j < nout) out[act_idx(j, tid)] = z + __ldg(bias + j);
                    }
                }
            } else
            for (int o0 = 0; o0 < npad; o0 += OCB) {
                // accumulators as pairs of adjacent outputs: [particle][output pair]
                unsigned long long tot[4 * R][2 * R], part[4 * R][2 * R];
#pragma unroll
                for (int a = 0; a < 4 * R; ++a)
#pragma unroll
                    for (int b = 0; b < 2 * R; ++b) { tot[a][b] = 0ull; part[a][b] = 0ull; }
                // weight slab of K chunk c: global -> shared by cp.async into buffer c & 1 while chunk c - 1 is being
                // multiplied; every thread moves PER 16-byte pieces (rows past K are not fetched and not read)
                constexpr int RP = OCB / 4;                              // 16-byte pieces per slab row
                constexpr int PER = KCH * RP / NT;
                static_assert(PER * NT == KCH * RP && NT % RP == 0 && KCH % 16 == 0 && 32 % KCH == 0, "slab pieces must divide over the threads");
                const float* wsrc = Wt + (size_t)(tid / RP) * npad + o0 + 4 * (tid % RP);
                const size_t ustep = (size_t)(NT / RP) * npad;
                auto fetch = [&](int k0, int buf) {
                    const float* s0 = wsrc + (size_t)k0 * npad;
                    const uint32_t d0 = ws_addr + (uint32_t)(buf * KCH * OCB * 4 + tid * 16);
#pragma unroll
                    for (int u = 0; u < PER; ++u)
                        if (k0 + tid / RP + u * (NT / RP) < K)
                            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d0 + u * NT * 16),
                                         "l"(s0 + u * ustep) : "memory");
                    asm volatile("cp.async.commit_group;" ::: "memory");
                };
                // one k step: R float4 of the activation row, R float4 of the weight row, (4R)^2 FFMA
                // ap = first row of a span that starts at a multiple of 16: the swizzle class of row k is (k >> 2) & 3
                auto lda = [&](const float* ap, int k, float4 (&av)[R]) {
#pragma unroll
                    for (int r = 0; r < R; ++r)
                        av[r] = *reinterpret_cast<const float4*>(ap + k * TP + pgx(k >> 2) + r * (TP / R));
                };
                auto ldw = [&](const float* wp, int k, float4 (&wv)[R]) {
#pragma unroll
                    for (int r = 0; r < R; ++r) wv[r] = *reinterpret_cast<const float4*>(wp + k * OCB + r * (OCB / R));
                };
                auto mac = [&](const float4 (&av)[R], const float4 (&wv)[R]) {
#pragma unroll
                    for (int ra = 0; ra < R; ++ra) {
                        const float a4[4] = {av[ra].x, av[ra].y, av[ra].z, av[ra].w};
#pragma unroll
                        for (int rb = 0; rb < R; ++rb) {
                            const unsigned long long w01 = pk2(wv[rb].x, wv[rb].y), w23 = pk2(wv[rb].z, wv[rb].w);
#pragma unroll
                            for (int a = 0; a < 4; ++a) {
                                const unsigned long long aa = pk2(a4[a], a4[a]);
                                part[4 * ra + a][2 * rb] = fma2(aa, w01, part[4 * ra + a][2 * rb]);
                                part[4 * ra + a][2 * rb + 1] = fma2(aa, w23, part[4 * ra + a][2 * rb + 1]);
                            }
                        }
                    }
                };
                fetch(0, c & 1);          // c runs on over output blocks and layers: buffer c & 1 was last read in
                                          // chunk c - 2, which every warp has left (barrier of chunk c - 1)
                for (int k0 = 0; k0 < K; k0 += KCH, ++c) {
                    const int kk = min(KCH, K - k0);
                    asm volatile("cp.async.wait_all;" ::: "memory");
                    __syncthreads();          // slab c visible; slab c - 1 consumed by every warp; layer input complete
                    if (k0 + KCH < K) fetch(k0 + KCH, (c + 1) & 1);
                    const float* __restrict__ ap = in + (size_t)k0 * TP;
                    const float* __restrict__ wp = Ws + (c & 1) * (KCH * OCB) + 4 * og;
                    if (kk == KCH) {
                        // operands of step k + 1 are loaded before the FFMAs of step k (the shared-memory latency
                        // was exposed with three warps per scheduler: profiles/r1_fp32.md); 16 steps per unrolled body
#pragma unroll 1
                        for (int h = 0; h < KCH / 16; ++h) {
                            const float* aph = ap + h * 16 * TP;
                            const float* wph = wp + h * 16 * OCB;
                            float4 av[R], wv[R];
                            lda(aph, 0, av); ldw(wph, 0, wv);
#pragma unroll
                            for (int k = 0; k < 16; ++k) {
                                float4 an[R], wn[R];
                                if (k + 1 < 16) { lda(aph, k + 1, an); ldw(wph, k + 1, wn); }
                                mac(av, wv);
                                if (k + 1 < 16) {
#pragma unroll
                                    for (int r = 0; r < R; ++r) { av[r] = an[r]; wv[r] = wn[r]; }
                                }
                            }
                        }
                    } else {
                        for (int k = 0; k < kk; ++k) {
                            float4 av[R], wv[R];
                            lda(ap, k, av); ldw(wp, k, wv);
                            mac(av, wv);
                        }
                    }
                    // partial sums of each 32-wide K span are formed separately and then added (shorter rounding chains)
                    if (((k0 / KCH) & (32 / KCH - 1)) == 32 / KCH - 1 || k0 + KCH >= K) {
#pragma unroll
                        for (int a = 0; a < 4 * R; ++a)
#pragma unroll
                            for (int b = 0; b < 2 * R; ++b) { tot[a][b] = add2(tot[a][b], part[a][b]); part[a][b] = 0ull; }
                    }
                }
#pragma unroll
                for (int rb = 0; rb < R; ++rb) {
                    const float4 bv = __ldg(reinterpret_cast<const float4*>(bias + o0 + rb * (OCB / R)) + og);
                    const float b4[4] = {bv.x, bv.y, bv.z, bv.w};
#pragma unroll
                    for (int b = 0; b < 4; ++b) {
#pragma unroll
                        for (int ra = 0; ra < R; ++ra) {
                            float r[4];
#pragma unroll
                            for (int a = 0; a < 4; ++a) {
                                float t0, t1;
                                unpk2(tot[4 * ra + a][2 * rb + (b >> 1)], t0, t1);
                                const float z = ((b & 1) ? t1 : t0) + b4[b];
                                r[a] = last ? z : hb_activate<ACT, false>(z, slope);
                            }
                            // rows o0 + rb OCB/R + 4 og + b: swizzle class og & 3 (o0 and OCB / R are multiples of 16)
                            *reinterpret_cast<float4*>(out + (size_t)(o0 + rb * (OCB / R) + 4 * og + b) * TP +
                                                       ra * (TP / R) + pgx_out) = make_float4(r[0], r[1], r[2], r[3]);
                        }
                    }
                }
            }
            float* tmp = in; in = out; out = tmp;
        }
        __syncthreads();
        if (tid < TP) {
            const size_t i = i0 + tid;
            if (i < n) {
                float w[6];
#pragma unroll
                for (int j = 0; j < 6; ++j) w[j] = in[act_idx(j, tid)];
                float x, px, y, py, t, pt;
                hb_sur_epilogue(sd, w, x, px, y, py, t, pt);
                p.v[0][i] = x; p.v[1][i] = px; p.v[2][i] = y; p.v[3][i] = py; p.v[4][i] = t; p.v[5][i] = pt;
                if (MOM) acc.add(sd.mom_pivot, x, px, y, py, t, pt);
            }
        }
    }
    if (MOM) {
        __syncthreads();
        hb_block_reduce_moments(acc, red, partials + blockIdx.x, tid, NT, 1);
    }
}

template <int TP, bool MOM, int R, int OCB, int KCH>
static cudaError_t launch_tp(const HbParticles& p, size_t n, const HbSurDev& sd, int hmax, double* partials,
                             int grid, bool prepare, cudaStream_t s) {
    constexpr int NT = (TP / (4 * R)) * (OCB / (4 * R));
    const size_t smem = ((size_t)2 * hmax * TP + 2 * KCH * OCB) * sizeof(float) + (NT / 32) * HB_NMOM * sizeof(double);
#define HB_LAUNCH_ACT(A)                                                                                         \
    {                                                                                                            \
        if (prepare)                                                                                             \
            return cudaFuncSetAttribute(hb_sur_fp32_kernel<TP, A, MOM, R, OCB, KCH>,                             \
                                        cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);                 \
        hb_sur_fp32_kernel<TP, A, MOM, R, OCB, KCH><<<grid, NT, smem, s>>>(p, n, sd, hmax, partials);            \
    }
    switch (sd.act) {
    case 0: HB_LAUNCH_ACT(0) break;
    case 1: HB_LAUNCH_ACT(1) break;
    case 2: HB_LAUNCH_ACT(2) break;
    default: HB_LAUNCH_ACT(3) break;
    }
#undef HB_LAUNCH_ACT
    return cudaGetLastError();
}

// HB_FP32_TP=16|32|64 : test / tuning hook, read by hb_lattice_finalize only (stored in the stage as fp32_tp): forces the
// 4 x 4 register-tile shape with that many particles per block
int hb_fp32_env_tp(void) {
    const char* force = getenv("HB_FP32_TP");
    return force ? atoi(force) : 0;
}

cudaError_t hb_launch_sur_fp32(const HbParticles& p, size_t n, const HbSurDev& sd, double* partials,
                               int* nblocks_out, int sm_count, bool prepare, cudaStream_t s) {
    int hmax = 64;
    for (int l = 0; l < sd.n_linear; ++l) hmax = hmax > sd.npad32[l] ? hmax : sd.npad32[l];
    // 8 x 8 register tiles (R = 2), 64 particles per block.  128 < hmax <= 256: 256-wide output blocks, 256 threads,
    // 32-row weight slabs, one block per SM (192 KB).  hmax = 128: 128-wide output blocks, 128 threads, two blocks per
    // SM (80 KB each).  Every layer that runs through the blocked loop must be padded to a multiple of the block width.
    const int force = sd.fp32_tp;
    const bool classic = force != 0 && force != 128;   // testing: force the 4 x 4 shapes
    auto blocked_multiple_of = [&](int m) {
        for (int l = 0; l < sd.n_linear; ++l) {
            const bool narrow_last = (l == sd.n_linear - 1) && sd.widths[l + 1] <= 8;
            if (!narrow_last && sd.npad32[l] % m != 0) return false;
        }
        return true;
    };
    const bool mom = partials != nullptr;
    const bool wide256 = !classic && hmax == 256 && blocked_multiple_of(256);
    const bool wide128 = !classic && hmax == 128 && blocked_multiple_of(128);
    if (wide256 || wide128) {
        const size_t ntiles = (n + 63) / 64;
        size_t g = (size_t)sm_count * (wide128 ? 2 : 1);
        if (g > ntiles) g = ntiles;
        if (g < 1) g = 1;
        if (nblocks_out) *nblocks_out = (int)g;
        if (wide256)
            return mom ? launch_tp<64, true, 2, 256, 32>(p, n, sd, hmax, partials, (int)g, prepare, s)
                       : launch_tp<64, false, 2, 256, 32>(p, n, sd, hmax, partials, (int)g, prepare, s);
        return mom ? launch_tp<64, true, 2, 128, 16>(p, n, sd, hmax, partials, (int)g, prepare, s)
                   : launch_tp<64, false, 2, 128, 16>(p, n, sd, hmax, partials, (int)g, prepare, s);
    }
    // 4 x 4 tiles: two activation buffers of hmax x TP floats beside the weight slabs; several blocks per SM when they
    // fit (independent blocks hide each other's barriers and slab loads): hmax 256 -> TP 32, 72 KB, 3 blocks/SM
    int tp = hmax <= 128 ? 64 : (hmax <= 768 ? 32 : 16);
    if (force) tp = force == 64 && hmax <= 384 ? 64 : (force == 16 ? 16 : (hmax <= 768 ? 32 : 16));
    const size_t smem_blk = ((size_t)2 * hmax * tp + 2 * KC * OC) * sizeof(float) + 1024;
    int per_sm = (int)((227 * 1024) / smem_blk);
    if (per_sm < 1) per_sm = 1;
    if (per_sm > 4) per_sm = 4;
    const size_t ntiles = (n + tp - 1) / tp;
    size_t g = (size_t)sm_count * per_sm;
    if (g > ntiles) g = ntiles;
    if (g < 1) g = 1;
    const int grid = (int)g;
    if (nblocks_out) *nblocks_out = grid;
    if (tp == 64) return mom ? launch_tp<64, true, 1, OC, KC>(p, n, sd, hmax, partials, grid, prepare, s) : launch_tp<64, false, 1, OC, KC>(p, n, sd, hmax, partials, grid, prepare, s);
    if (tp == 32) return mom ? launch_tp<32, true, 1, OC, KC>(p, n, sd, hmax, partials, grid, prepare, s) : launch_tp<32, false, 1, OC, KC>(p, n, sd, hmax, partials, grid, prepare, s);
    return mom ? launch_tp<16, true, 1, OC, KC>(p, n, sd, hmax, partials, grid, prepare, s) : launch_tp<16, false, 1, OC, KC>(p, n, sd, hmax, partials, grid, prepare, s);
}
