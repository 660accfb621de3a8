/*
 * hb.h -- C ABI of libhb.so: B200-native (sm_100a) hybrid conventional/surrogate beamline push.
 *
 * Method: Sandberg et al., "Synthesizing Particle-in-Cell Simulations Through Learning and GPU
 * Computing for Hybrid Particle Accelerator Beamlines", PASC'24 (arXiv 2402.17248).
 * Citations "P:NN" are lines of PAPER.md; "R1..R10" / "G1..G17" are the readings in DESIGN.md.
 *
 * What one hb_push computes (every element, conventional or surrogate, is a per-particle
 * map R^6 -> R^6, so the whole push is data-parallel over particles): an N-particle bunch, resident
 * in device memory as six fp32 arrays (x, px, y, py, t, pt; s-based coordinates relative to a
 * reference particle, R1), is pushed IN PLACE through the lattice:
 *   - runs of conventional elements (drift R2, thick quadrupole R3, sector bend R4)
 *     are fused into one pass over HBM per run;
 *   - a surrogate stage is  [s->t conversion, R6]  ->  per-coordinate normalisation
 *     (R8)  ->  MLP  F = L_l o sigma o ... o sigma o L_0  (Eq. 1-3, R9)  ->
 *     de-normalisation  ->  [reference update R7, t->s conversion R6];
 *   - a monitor records the bunch moments (R10) of the current state.
 *
 * Everything is extern "C"; no C++ or torch types cross the boundary.  Particle arrays and the
 * moments buffer are DEVICE pointers borrowed for the duration of the enqueued work; every other
 * pointer is a HOST pointer that is deep-copied before the call returns.  All device work is
 * enqueued on the caller's stream; no entry point synchronises the device except
 * hb_lattice_finalize (uploads) and hb_lattice_destroy.  There is no CPU fallback: without a
 * usable sm_100 device the calls fail with HB_ERR_CUDA / HB_ERR_UNSUPPORTED.
 */
#ifndef HB_H
#define HB_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct hb_lattice hb_lattice; /* opaque; owned by the library */

typedef enum {
    HB_OK = 0,
    HB_ERR_INVALID_ARG = 1, /* NULL / misaligned / aliasing pointers, non-finite or out-of-range values */
    HB_ERR_STATE = 2,       /* adding to a finalized lattice, pushing a non-finalized one */
    HB_ERR_ALLOC = 3,       /* host or device allocation failed */
    HB_ERR_CUDA = 4,        /* a CUDA runtime call or a kernel launch failed (see hb_last_error) */
    HB_ERR_UNSUPPORTED = 5  /* valid request the library has no kernel for (never a CPU fallback) */
} hb_status;

/* Conventional elements (formulas R2-R4).  MONITOR is the identity map that emits one
 * 27-double moment record (R10) and splits runs (R5, G17).  PLENS: thick axisymmetric linear (plasma) lens
 * (R3b): x'' = -k x and y'' = -k y, k > 0 focuses both planes; the paper sets k from the
 * moments of the previous monitor with an expression it does not print -- here the caller supplies k
 * (read the record, build the next lattice).
 * DRIFT_EXACT: drift without the paraxial expansion of R2 (R2x: x += L px/pz, t += L((1/beta0 - pt)/pz - 1/beta0),
 * pz = sqrt(1 - 2 pt/beta0 + pt^2 - px^2 - py^2)); non-linear, so a run that contains one is always applied
 * element by element in fp64 registers (the SEQUENTIAL kernel), whatever the run mode.
 * QUAD_CHROMATIC (R3x): thick quadrupole with momentum-dependent focusing, omega^2 = k/(1+delta), and the betatron
 * term in the time of flight.  MULTIPOLE (R5x): thin kick, added with hb_lattice_add_multipole.  Both non-linear. */
typedef enum { HB_ELEM_DRIFT = 0, HB_ELEM_QUAD = 1, HB_ELEM_SBEND = 2, HB_ELEM_MONITOR = 3, HB_ELEM_PLENS = 5,
               HB_ELEM_DRIFT_EXACT = 6, HB_ELEM_QUAD_CHROMATIC = 7, HB_ELEM_MULTIPOLE = 8 } hb_elem_kind;

/* Activation sigma of Eq. 3: identity; ReLU Eq. 1; PReLU Eq. 2, one learned
 * slope per activation layer (G9); tanh (the "sigmoidal function" of P:90; BASELINE configs 1,4,5). */
typedef enum { HB_ACT_IDENTITY = 0, HB_ACT_RELU = 1, HB_ACT_PRELU = 2, HB_ACT_TANH = 3 } hb_act;

/* Arithmetic of the MLP layers.  FP32: CUDA-core FFMA.  BF16/F16/TF32: tcgen05 tensor cores with
 * operands rounded to that type and fp32 accumulation in TMEM.  Shapes: BF16/F16 any hidden widths <= 256
 * whose 16-bit weights fit in shared memory (resident kernels), else equal hidden widths <= 512 (weights
 * streamed from L2), else equal hidden widths <= 1024 (one launch per layer, activations through a 2-4 GB global
 * scratch allocated at finalize; bunches up to 3.3e7 particles per push); TF32 (half the tensor rate): at least one
 * hidden layer, equal hidden widths <= 256.
 * Anything else: hb_lattice_finalize returns HB_ERR_UNSUPPORTED -- never a slower fallback.
 * ACCURACY against the fp64 definition, max |error| over the bunch in units of the output coordinate's std (measured on
 * the synthetic random networks of BASELINE.json; trained networks are smoother):
 *   FP32  <= 1e-5 (4.5e-6 on 6-256^3-6; a 6-512^4-6 tanh net sits at the format's own level, 1e-5).
 *   F16   4e-3 .. 1.5e-2: the 16-bit mode that MEETS the 2e-2 bound of the tensor-core path; same instruction and rate
 *         as BF16.  RANGE: an fp16 operand overflows at 65504 -- a hidden activation above that becomes +inf (ReLU,
 *         PReLU and identity activations are unbounded; tanh is not).  The inputs are normalised to O(1) (R8) and
 *         He / Xavier-scaled layers keep activations O(1..10); a net whose hidden activations can exceed 6e4 needs
 *         BF16, TF32 or FP32.
 *   TF32  5e-3 .. 1.8e-2 (10 explicit significand bits like F16, fp32 range; half the rate).
 *   BF16  4e-2 .. 1.4e-1: 8 significand bits; OUTSIDE the 2e-2 bound on these networks.  It is kept because the paper's
 *         configs name it and because it has fp32 range; it is a reported, NOT a conforming mode
 *         (tests/test_gpu_stagefed.py::test_plain_bf16_does_not_meet_the_north_star_bound states the miss). */
typedef enum { HB_PREC_FP32 = 0, HB_PREC_BF16 = 1, HB_PREC_F16 = 2, HB_PREC_TF32 = 3 } hb_prec;

/* Coordinates the surrogate was trained in.  HB_COORD_S: the net sees (x,px,y,py,t,pt) as is.
 * HB_COORD_T: the net sees fixed-time coordinates (x,y,z,ux,uy,uz), momenta in units of mc
 * (P:60-62); the library converts s->t before and t->s after (R6) and moves the
 * reference particle to the stage's output energy (R7; "about 7 GeV energy gain per stage"). */
typedef enum { HB_COORD_S = 0, HB_COORD_T = 1 } hb_coord;

/* How a run of conventional elements is applied.
 * COMPOSED: the run's elements are concatenated on the host in fp64 into one 6x6 map (standard
 *   transfer-matrix concatenation), rounded once to fp32 and applied in one HBM pass.
 * SEQUENTIAL: the element list is applied one by one in fp64 registers, one rounding at the store.
 * SEQUENTIAL_FP32: as SEQUENTIAL but in fp32 registers (literal reading of "fp32, element parameters
 *   in constant or shared memory").  Every element rounds its coefficients and its result to fp32 (~3e-8 relative
 *   each, partly systematic): measured max |error| / std against the fp64 definition is 1.1e-6 after ONE FODO cell
 *   (5 elements) -- already above the 1e-6 bound of the element maps -- and 2e-5 .. 5e-5 after 500 elements
 *   (tests/test_gpu_parity.py::test_sequential_fp32_reported_not_bounded holds it to 2e-4).  A reported mode, not a
 *   conforming one: COMPOSED and SEQUENTIAL meet 1e-6 at any run length. */
typedef enum { HB_RUN_COMPOSED = 0, HB_RUN_SEQUENTIAL = 1, HB_RUN_SEQUENTIAL_FP32 = 2 } hb_run_mode;

/* One surrogate stage (all pointers HOST pointers, deep-copied by hb_lattice_add_surrogate). */
typedef struct {
    int n_linear;            /* l+1 linear maps L_0..L_l; >= 1                                   */
    const int *widths;       /* n_linear+1 entries: 6, H_1, ..., H_l, 6  (n = m = 6); 1<=H<=1024 */
    const float *const *W;   /* n_linear matrices A_i, row-major [out][in]                               */
    const float *const *b;   /* n_linear bias vectors b_i, [out]                                          */
    hb_act act;              /* the same sigma after L_0..L_{l-1}, none after L_l (G7)         */
    const float *prelu_a;    /* HB_ACT_PRELU: n_linear-1 slopes (one per activation layer, G9); else NULL */
    double in_mean[6], in_std[6];   /* input normalisation  v^ = (v - mean)/std  (R8), std > 0    */
    double out_mean[6], out_std[6]; /* output de-normalisation w = w^ * std + mean        */
    hb_coord coord;
    double ref_bg_out;       /* COORD_T: (beta gamma) of the reference after the stage; NaN = evaluate the
                                net on the reference input (0,0,0,0,0,(beta gamma)_in) in fp64 on the host
                                at finalize and take component uz (R7)                                    */
    double ref_z_out;        /* COORD_T: reference z after the stage, subtracted from every particle's z;
                                NaN = component z of the same host evaluation                            */
    hb_prec prec;
} hb_surrogate_desc;

/* Create an empty lattice for a reference particle of the given kinetic and rest energy [MeV] (R1:
 * gamma0 = 1 + T/mc^2).  Errors: NULL out, non-finite / non-positive energies -> INVALID_ARG. */
hb_status hb_lattice_create(double ref_kinetic_energy_MeV, double rest_energy_MeV, hb_lattice **out);

/* Append a conventional element.  length_m: DRIFT any finite value (negative allowed: the
 * drift(L) o drift(-L) identity test needs it); QUAD, SBEND >= 0; MONITOR ignored.
 * param: QUAD k [1/m^2] (k > 0 focuses x, R3); PLENS k [1/m^2] (k > 0 focuses x and y, R3b); SBEND bend angle
 * [rad], signed (R4); else ignored.
 * Errors: finalized lattice -> STATE; non-finite or negative QUAD/SBEND length -> INVALID_ARG. */
hb_status hb_lattice_add_element(hb_lattice *lat, hb_elem_kind kind, double length_m, double param);

/* Change length and parameter of element `index` (0-based position in the order of the add calls; monitors and
 * surrogate stages count) -- the elements of a beamline are "programmable at run time", and the paper's
 * optimisation (Nelder-Mead over lens position and strength, one tracking run per evaluation) changes two or
 * three of them between pushes.  Allowed before and after hb_lattice_finalize; the element keeps its kind.  On a
 * finalized lattice only the run that holds the element is rebuilt (fp64 concatenation of its maps on the host, R5);
 * surrogate weights, records and scratch are untouched.  The call synchronises the lattice's device (the element table
 * of sequential runs is device-resident), so it orders itself after every push enqueued before it; a CUDA graph
 * captured earlier keeps the old maps and must be re-captured.
 * Errors: index out of range, or a monitor / surrogate / multipole element -> INVALID_ARG; values as in
 * hb_lattice_add_element. */
hb_status hb_lattice_set_element(hb_lattice *lat, int index, double length_m, double param);

/* Append a thin multipole kick (R5x) of order m (1 dipole, 2 quadrupole, 3 sextupole, ... <= 8) with integrated normal
 * and skew strengths kn, ks [m^-(m-1)]:  px - i py -= (kn + i ks)(x + i y)^(m-1)/(m-1)!.  Non-linear for m > 2: the run
 * that holds it is applied element by element in fp64 registers.  Errors as hb_lattice_add_element. */
hb_status hb_lattice_add_multipole(hb_lattice *lat, int order, double kn, double ks);

/* Append a surrogate stage; deep-copies every host array of *desc.
 * Errors: widths[0] != 6 or widths[last] != 6, H outside [1,1024], std <= 0, non-finite values,
 * PRELU without slopes -> INVALID_ARG; finalized lattice -> STATE. */
hb_status hb_lattice_add_surrogate(hb_lattice *lat, const hb_surrogate_desc *desc);

/* Choose how conventional runs are applied (default HB_RUN_COMPOSED).  Before finalize only. */
hb_status hb_lattice_set_run_mode(hb_lattice *lat, hb_run_mode mode);

/* Nominal centroid of the incoming bunch in (x,px,y,py,t,pt), HOST, 6 doubles; default all zero (a bunch centred on
 * the reference particle).  The library tracks it through the lattice on the host (run matrices; a surrogate stage
 * sends it to its out_mean) and uses the tracked value as the pivot of the moment sums of every monitor (R10): sums of
 * (v - pivot) are accumulated and the pivot is added back to the means, so a record does not depend on it beyond
 * rounding -- it only keeps E[v^2] - E[v]^2 well conditioned for a bunch far off axis with a small spread.  Allowed
 * before and after finalize (host arithmetic only).  Errors: NULL / non-finite -> INVALID_ARG. */
hb_status hb_lattice_set_centroid(hb_lattice *lat, const double *centroid6);

/* Split the element list into segments (maximal runs of conventional elements; single surrogate
 * stages; monitors), track the reference particle (R7), compose runs in fp64, pack the weights into
 * the tensor-core operand layout, upload constants and allocate all scratch on `cuda_device`.
 * Synchronises that device's uploads.  Errors: no such device / not sm_100 -> CUDA / UNSUPPORTED;
 * a surrogate shape the library has no kernel for -> UNSUPPORTED; second call -> STATE. */
hb_status hb_lattice_finalize(hb_lattice *lat, int cuda_device);

/* Number of MONITOR elements (= moment records one push produces). */
hb_status hb_lattice_num_monitors(const hb_lattice *lat, int *out);

/* Number of kernel launches one hb_push / hb_push_moments of n_particles enqueues (launch accounting): one per run and
 * per surrogate stage -- a layered wide-net stage (hidden widths 513..1024) is one per linear layer and chunk of 2^20
 * particles -- plus one finalize per fused monitor and two per standalone monitor.  n_particles = 0: no launch. */
hb_status hb_lattice_num_launches(const hb_lattice *lat, int with_moments, size_t n_particles, int *out);

/* (beta gamma) of the reference particle after the last element (valid after finalize). */
hb_status hb_lattice_ref_bg_out(const hb_lattice *lat, double *out);

/* Push n particles through the lattice in place.  x..pt: six DEVICE arrays of n floats each, 16-byte
 * aligned, pairwise non-overlapping; borrowed until the enqueued work completes.  n >= 0 (0 is a
 * no-op).  cuda_stream: a cudaStream_t (NULL = legacy default stream).  Returns after enqueueing;
 * MONITOR elements are skipped.  Errors: not finalized -> STATE; NULL / misaligned / overlapping
 * arrays -> INVALID_ARG; launch failure -> CUDA.
 * ONE PUSH IN FLIGHT PER LATTICE: a lattice owns one buffer of moment partials and (wide nets) one activation scratch,
 * allocated at finalize and reused by every push (nothing is allocated per push).  Pushes of the same lattice are safe
 * back to back on ONE stream; pushes of the same lattice on DIFFERENT streams (hb_push, hb_push_moments, hb_push_host,
 * hb_push_candidates) must be ordered by the caller (an event between them), or use one lattice object per stream --
 * the device-resident state of a lattice is its weights (<= a few MB) and that scratch. */
hb_status hb_push(hb_lattice *lat, float *x, float *px, float *y, float *py, float *t, float *pt,
                  size_t n, void *cuda_stream);

/* As hb_push, and writes one record of 27 doubles per MONITOR to d_moments (DEVICE, 8-byte aligned,
 * num_monitors x 27): [0..5] means of (x,px,y,py,t,pt); [6..26] upper triangle, row-major, of the
 * centred second moments with uniform weights and 1/N (R10, G11; sigma_x, eps_x of P:138, P:146
 * follow from these).  Moments are accumulated in fp64 inside the kernel that produces the state
 * (or by a standalone pass when a monitor has no producing kernel) and finished by a fixed-order
 * reduction: deterministic, no floating-point atomics.  n = 0 writes NaN records. */
hb_status hb_push_moments(hb_lattice *lat, float *x, float *px, float *y, float *py, float *t, float *pt,
                          size_t n, double *d_moments, void *cuda_stream);

/* Push a bunch that lives in HOST memory (six arrays of n floats; page-locked memory makes the copies asynchronous).
 * The library stages it through device buffers it owns (allocated at the first call, kept until destroy) in `chunks`
 * pieces through a three-stage pipeline (internal copy-in, compute and copy-out streams, three staging slots): the
 * host->device copy of piece i+1 and the device->host copy of piece i-1 overlap the kernels of piece i.  Every particle goes through exactly the kernels of hb_push_moments; the
 * moment partials of all pieces are summed by the same finalize kernel, so each record is the record of the whole
 * bunch.  In place: the host arrays hold the result on return.  h_moments: host, num_monitors x 27 doubles, or NULL.
 * chunks: 1..8.  SYNCHRONOUS (returns when the result is in host memory); n = 0 is a no-op (NaN records).
 * Errors: as hb_push_moments (the 16-byte alignment requirement does not apply to host arrays). */
hb_status hb_push_host(hb_lattice *lat, float *x, float *px, float *y, float *py, float *t, float *pt,
                       size_t n, double *h_moments, int chunks);

/* K candidate settings of one transport section over the SAME resident bunch, in one pass (the
 * paper optimises position and strength of the lens in every gap between stages, 2 (N_stage - 1) = 28 parameters,
 * stage by stage with Nelder-Mead, one tracking run per evaluation -- and every evaluation of one gap starts from the
 * same bunch).  elem_index: n_set elements (positions in the order of the add calls) of ONE run of conventional
 * elements; length_m, param: HOST, [n_candidates][n_set], the settings of those elements for candidate k (meaning and
 * validation as hb_lattice_set_element).  x..pt: the bunch AS IT ENTERS THAT RUN (device, n floats each, 16-byte
 * aligned); it is only read.  The lattice itself is not changed.
 * d_moments: DEVICE, n_candidates x 27 doubles: record k = the moments (R10, layout of hb_push_moments) of the bunch
 * behind the run with candidate k's settings.
 * How: every candidate's run is concatenated on the host in fp64 into one 6x6 map M_k (R5), as hb_lattice_finalize
 * does; for a linear map the sample moments transform exactly (mean' = M mean, C' = M C M^T), so the bunch is read ONCE
 * (24 B per particle, the fused fp64 reduction of hb_moments) whatever n_candidates is, and one thread per candidate
 * does the 6x6 products in fp64: three launches per call.  The records are those of the exact image of the fp32 input;
 * a push of the same setting rounds every coordinate to fp32 once more, which moves second moments by <= 1e-7 relative.
 * Asynchronous on cuda_stream like hb_push (the host arrays are consumed before the call returns).  n = 0: NaN records.
 * Errors: not finalized -> STATE; elements not all in one run, a multipole, invalid values -> INVALID_ARG; a run that
 * holds a non-linear element (no composed map) -> UNSUPPORTED. */
hb_status hb_push_candidates(hb_lattice *lat, int n_candidates, int n_set, const int *elem_index, const double *length_m,
                             const double *param, const float *x, const float *px, const float *y, const float *py,
                             const float *t, const float *pt, size_t n, double *d_moments, void *cuda_stream);

/* Standalone moments of a bunch (R10).  pivot: 6 HOST doubles subtracted before accumulation (any
 * value near the bunch centre; NULL = zeros); the result does not depend on it beyond rounding.
 * d_out27: DEVICE, 27 doubles.  d_scratch: DEVICE scratch of hb_moments_scratch_bytes() bytes. */
hb_status hb_moments(const float *x, const float *px, const float *y, const float *py, const float *t,
                     const float *pt, size_t n, const double *pivot, double *d_out27, void *d_scratch,
                     void *cuda_stream);
size_t hb_moments_scratch_bytes(void);

/* hb_moments() for callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): the same two kernels, the same record (bit-identical), with the block-partials
 * scratch in a file-scope array of the library's device image -- 27 x 4736 doubles = 999 KB that every GPU which loads
 * libhb.so holds until the process exits.  The call allocates and frees NOTHING (no cudaMalloc / cudaFree, no allocating
 * library routine); the first call on a device looks the array's address up (cudaGetSymbolAddress, with that device
 * current -- make one call before starting a capture).  Runs on the CURRENT device, on cuda_stream, asynchronously.
 * Arguments as hb_moments(); n <= HB_MOMENTS_STATIC_MAX_N, else HB_ERR_INVALID_ARG (hb_last_error() names the limit);
 * NULL / misaligned arrays: HB_ERR_INVALID_ARG; a device other than compute capability 10.0: HB_ERR_UNSUPPORTED.
 * SHARED STATE: every call on a device uses the same array.  Nothing in it has to start at zero and nothing of the
 * previous call is read (each call overwrites the rows it reads), but two calls that overlap on the GPU (different
 * streams, no ordering between them) RACE: order them on one stream or with events. */
#define HB_MOMENTS_STATIC_MAX_N 268435456ull /* 2^28 particles: a 6.4 GB bunch */
hb_status hb_moments_static(const float *x, const float *px, const float *y, const float *py, const float *t,
                            const float *pt, size_t n, const double *pivot, double *d_out27, void *cuda_stream);
size_t hb_moments_static_max_particles(void); /* HB_MOMENTS_STATIC_MAX_N, for bindings */

/* Record of the union of two disjoint particle sets from their records (HOST arithmetic, no device needed):
 * the sharded-monitor step of a distributed bunch (every rank pushes its own particles; a monitor, P:138,
 * is over all of them).  rec_a / rec_b: HOST, 27 doubles each as hb_push_moments writes them (6 means, then the
 * 21 centred second moments with 1/N, upper triangle row-major); n_a, n_b: the particle counts behind them.
 *   mean = (n_a mean_a + n_b mean_b) / n,   C = (n_a C_a + n_b C_b) / n + (n_a n_b / n^2) d d^T,  d = mean_b - mean_a
 * (the pairwise update of the raw sums of R10, exact up to rounding).  A set with n = 0 contributes nothing (its
 * record may hold NaN); n_a = n_b = 0 writes NaN.  rec_out: HOST, 27 doubles, may alias rec_a or rec_b.
 * Errors: NULL pointer -> HB_ERR_INVALID_ARG. */
hb_status hb_moments_merge(const double *rec_a, unsigned long long n_a, const double *rec_b, unsigned long long n_b,
                           double *rec_out);

/* Optional per-segment device timing (observability; P:199 gives the paper's manual breakdown).  When on,
 * every push records a CUDA event before the first and after each segment's kernels on the caller's stream.
 * hb_lattice_get_timing synchronises on the last event of the most recent push and writes, for each of the
 * n segments (runs, surrogate stages, standalone monitors, in lattice order; a fused monitor's finalize is
 * counted with its segment), the elapsed milliseconds to ms_out[0..min(n,capacity)) and n to *n_out. */
hb_status hb_lattice_enable_timing(hb_lattice *lat, int on);
hb_status hb_lattice_get_timing(hb_lattice *lat, float *ms_out, int capacity, int *n_out);

/* Measured throughput of the pipes the kernels are bound by, on device `cuda_device` (synchronous, ~50 ms; no lattice
 * needed): out5[0] fp32 FMA [TFMA/s], out5[1] fp64 FMA [TFMA/s], out5[2] MUFU tanh.approx [T results/s],
 * out5[3] tcgen05.mma kind::f16 and out5[4] kind::tf32, M128 x N256, operands in shared memory, fp32 accumulate
 * [TFLOP/s].  Short kernels: burst rates of the pipes at the unloaded clock, not sustained power-limited figures.
 * Observability (P:199 reports the paper's own time breakdown): bench.py quotes the ALU-bound kernels and the tf32 mode
 * against these instead of datasheet unit counts.  Errors: NULL -> INVALID_ARG; no such device -> CUDA; not sm_100 ->
 * UNSUPPORTED. */
hb_status hb_device_peaks(int cuda_device, double *out5);

/* Destroy the lattice and free everything it owns (synchronises its device).  NULL is a no-op. */
hb_status hb_lattice_destroy(hb_lattice *lat);

const char *hb_status_string(hb_status s);
const char *hb_last_error(void); /* thread-local message of the last failing call on this thread */
const char *hb_version(void);

/* Which kernel a surrogate stage of this shape runs on (host-only query, no device needed; the same decision
 * hb_lattice_finalize takes): "fp32-ffma", "tcgen05-resident" (16-bit weights resident in shared memory),
 * "tcgen05-streamed" (weights streamed from L2; also every HB_PREC_TF32 stage), "tcgen05-layered" (hidden widths
 * 513..1024: one launch per layer, activations through a global scratch the lattice owns), or NULL when the shape has no
 * schedule (hb_lattice_finalize would return HB_ERR_UNSUPPORTED; reason in hb_last_error()).
 * widths: n_linear + 1 entries, 6, H_1, ..., 6.  The returned string is static. */
const char *hb_surrogate_kernel(hb_prec prec, int n_linear, const int *widths);

#ifdef __cplusplus
}
#endif
#endif /* HB_H */
