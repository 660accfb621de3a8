// hb_api.cu -- the C ABI of include/hb.h: lattice construction, reference tracking (R1, R7), fp64
// composition of conventional runs (R2-R5), weight packing, segment sequencing (row a7).
// Host code only; kernels live in hb_run.cu / hb_sur_fp32.cu / hb_sur_tc.cu.
#include <limits>
#include "../../include/hb.h"
#include "hb_internal.h"

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

namespace {

thread_local std::string g_err;

hb_status fail(hb_status s, const char* fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    g_err = buf;
    return s;
}

#define HB_CUDA(call)                                                                              \
    do {                                                                                           \
        cudaError_t e_ = (call);                                                                   \
        if (e_ != cudaSuccess) return fail(HB_ERR_CUDA, "%s: %s", #call, cudaGetErrorString(e_));  \
    } while (0)

struct Elem {
    int kind;        // hb_elem_kind, or 4 = surrogate
    double L, param;
    int sur;         // index into surrogates
    double p2 = 0.0; // MULTIPOLE: skew strength (L = order, param = normal strength)
};

bool is_conventional(int kind) {
    return kind <= HB_ELEM_SBEND || kind == HB_ELEM_PLENS || kind == HB_ELEM_DRIFT_EXACT ||
           kind == HB_ELEM_QUAD_CHROMATIC || kind == HB_ELEM_MULTIPOLE;
}
bool is_nonlinear(int kind) {
    return kind == HB_ELEM_DRIFT_EXACT || kind == HB_ELEM_QUAD_CHROMATIC || kind == HB_ELEM_MULTIPOLE;
}

struct SurHost {
    int n_linear;
    std::vector<int> widths;
    std::vector<std::vector<float>> W, b;
    int act;
    std::vector<float> prelu;
    double in_mean[6], in_std[6], out_mean[6], out_std[6];
    int coord;
    double ref_bg_out, ref_z_out;
    int prec;
};

enum SegType { SEG_RUN = 0, SEG_SUR = 1, SEG_MON = 2 };

struct Segment {
    int type;
    HbRunMap map;          // SEG_RUN composed
    int seq_off, seq_cnt;  // SEG_RUN sequential: range in d_seq
    int e_lo, e_hi;        // SEG_RUN: its elements are lat->elems[e_lo, e_hi)
    double bg;             // SEG_RUN: (beta gamma) of the reference inside the run
    bool nonlinear;        // SEG_RUN holds a non-linear element: no composed map, always the fp64 sequential kernel
    HbSurDev sd;           // SEG_SUR
    int sur;               // SEG_SUR: index into lat->surs
    double bg1, z1;        // SEG_SUR, COORD_T: outgoing reference (given or derived, R7)
    bool tc;               // SEG_SUR: tensor-core kernel
    int monitor;           // record index written after this segment, -1 = none
    double pivot[6];       // nominal centroid of the state behind this segment: pivot of its moment sums (a3)
};

// ---- fp64 6x6 helpers (transfer-matrix concatenation, R5) ---------------------------------
struct Mat6 { double m[6][6]; };

Mat6 mat_identity() {
    Mat6 r;
    for (int i = 0; i < 6; ++i)
        for (int j = 0; j < 6; ++j) r.m[i][j] = i == j ? 1.0 : 0.0;
    return r;
}

Mat6 mat_mul(const Mat6& a, const Mat6& b) {   // a * b
    Mat6 r;
    for (int i = 0; i < 6; ++i)
        for (int j = 0; j < 6; ++j) {
            double s = 0.0;
            for (int k = 0; k < 6; ++k) s += a.m[i][k] * b.m[k][j];
            r.m[i][j] = s;
        }
    return r;
}

// sin(x)/x and (1-cos x)/x without a branch on x == 0 in the result (series for tiny |x|)
double sinc_(double x) { return std::fabs(x) < 1e-6 ? 1.0 - x * x / 6.0 : std::sin(x) / x; }
double cosc_(double x) {   // (1 - cos x)/x = sin^2(x/2)/(x/2)
    const double h = 0.5 * x;
    return std::sin(h) * sinc_(h);
}

// element matrix in the lattice's s-coordinates (x,px,y,py,t,pt); bg = (beta gamma) of the reference
Mat6 elem_matrix(const Elem& e, double bg) {
    Mat6 M = mat_identity();
    const double L = e.L;
    const double r56 = L / (bg * bg);
    if (e.kind == HB_ELEM_DRIFT || e.kind == HB_ELEM_DRIFT_EXACT) {   // (exact drift: its linearisation, unused)
        M.m[0][1] = L; M.m[2][3] = L; M.m[4][5] = r56;
    } else if (e.kind == HB_ELEM_MULTIPOLE) {
        // identity (thin; the run it sits in is never composed)
    } else if (e.kind == HB_ELEM_QUAD || e.kind == HB_ELEM_PLENS || e.kind == HB_ELEM_QUAD_CHROMATIC) {
        const double k = e.param, w = std::sqrt(std::fabs(k)), ph = w * L;
        // focusing plane: [cos, sin/w; -w sin, cos]; defocusing: [cosh, sinh/w; w sinh, cosh]
        double f[4], d[4];
        f[0] = std::cos(ph); f[1] = L * sinc_(ph); f[2] = -w * std::sin(ph); f[3] = f[0];
        d[0] = std::cosh(ph);
        d[1] = ph < 1e-6 ? L * (1.0 + ph * ph / 6.0) : std::sinh(ph) / w;
        d[2] = w * std::sinh(ph); d[3] = d[0];
        const double* X = k >= 0 ? f : d;
        const double* Y = e.kind == HB_ELEM_PLENS ? X : (k >= 0 ? d : f);     // lens: same sign in both planes (R3b)
        M.m[0][0] = X[0]; M.m[0][1] = X[1]; M.m[1][0] = X[2]; M.m[1][1] = X[3];
        M.m[2][2] = Y[0]; M.m[2][3] = Y[1]; M.m[3][2] = Y[2]; M.m[3][3] = Y[3];
        M.m[4][5] = r56;
    } else if (e.kind == HB_ELEM_SBEND) {
        const double th = e.param;
        const double g = std::sqrt(1.0 + bg * bg), b0 = bg / g;
        const double s = std::sin(th), c = std::cos(th);
        const double rs = L * sinc_(th);        // rho sin(theta)
        const double rc = L * cosc_(th);        // rho (1 - cos theta)
        const double h_s = th == 0.0 ? 0.0 : s * th / L;   // sin(theta)/rho
        M.m[0][0] = c;    M.m[0][1] = rs;  M.m[0][5] = -rc / b0;
        M.m[1][0] = -h_s; M.m[1][1] = c;   M.m[1][5] = -s / b0;
        M.m[2][3] = L;
        M.m[4][0] = s / b0; M.m[4][1] = rc / b0;
        // rho(-theta + sin(theta)/b0^2) = -L + rs/b0^2 = L(1-b0^2)/b0^2 - (L - rs)/b0^2 ; 1-b0^2 = 1/g^2
        M.m[4][5] = L / (bg * bg) - (L - rs) / (b0 * b0);
    }
    return M;
}

HbSeqElem seq_elem(const Elem& e, double bg) {
    const Mat6 M = elem_matrix(e, bg);
    HbSeqElem s;
    std::memset(&s, 0, sizeof s);
    s.kind = e.kind == HB_ELEM_PLENS ? (int)HB_ELEM_QUAD : e.kind;   // the device applies a lens as two 2x2 planes + t
    if (e.kind == HB_ELEM_QUAD_CHROMATIC) {
        s.kind = 4;
        s.a[0] = e.L; s.a[1] = e.param; s.a[2] = std::sqrt(1.0 + bg * bg) / bg;
    } else if (e.kind == HB_ELEM_MULTIPOLE) {
        s.kind = 5;
        const int m = (int)e.L;
        double fact = 1.0;
        for (int j = 2; j < m; ++j) fact *= j;
        s.a[0] = e.param / fact; s.a[1] = e.p2 / fact; s.a[2] = (double)m;
    } else if (e.kind == HB_ELEM_DRIFT_EXACT) {
        s.kind = 3;
        s.a[0] = e.L; s.a[1] = std::sqrt(1.0 + bg * bg) / bg;      // 1/beta0
    } else if (e.kind == HB_ELEM_DRIFT) {
        s.a[0] = e.L; s.a[1] = M.m[4][5];
    } else if (e.kind == HB_ELEM_QUAD || e.kind == HB_ELEM_PLENS) {
        s.a[0] = M.m[0][0]; s.a[1] = M.m[0][1]; s.a[2] = M.m[1][0]; s.a[3] = M.m[1][1];
        s.a[4] = M.m[2][2]; s.a[5] = M.m[2][3]; s.a[6] = M.m[3][2]; s.a[7] = M.m[3][3];
        s.a[8] = M.m[4][5];
    } else {
        s.a[0] = M.m[0][0]; s.a[1] = M.m[0][1]; s.a[2] = M.m[1][0]; s.a[3] = M.m[1][1];
        s.a[4] = M.m[0][5]; s.a[5] = M.m[1][5]; s.a[6] = M.m[2][3];
        s.a[7] = M.m[4][0]; s.a[8] = M.m[4][1]; s.a[9] = M.m[4][5];
    }
    return s;
}

double act_host(double z, int act, double a) {
    switch (act) {
    case HB_ACT_RELU: return z >= 0 ? z : 0.0;
    case HB_ACT_PRELU: return z >= 0 ? z : a * z;
    case HB_ACT_TANH: return std::tanh(z);
    default: return z;
    }
}

// fp64 host evaluation of the net on one vector (R7: reference particle through a COORD_T stage)
void mlp_host(const SurHost& s, const double in[6], double out[6]) {
    std::vector<double> h(in, in + 6), g;
    for (int j = 0; j < 6; ++j) h[j] = (in[j] - s.in_mean[j]) / s.in_std[j];
    for (int l = 0; l < s.n_linear; ++l) {
        const int fin = s.widths[l], fout = s.widths[l + 1];
        g.assign(fout, 0.0);
        for (int o = 0; o < fout; ++o) {
            double acc = 0.0;
            for (int k = 0; k < fin; ++k) acc += (double)s.W[l][(size_t)o * fin + k] * h[k];
            acc += (double)s.b[l][o];
            if (l < s.n_linear - 1) acc = act_host(acc, s.act, s.act == HB_ACT_PRELU ? (double)s.prelu[l] : 0.0);
            g[o] = acc;
        }
        h.swap(g);
    }
    for (int j = 0; j < 6; ++j) out[j] = h[j] * s.out_std[j] + s.out_mean[j];
}

void split_hi_lo(double v, float& hi, float& lo) {
    hi = (float)v;
    lo = (float)(v - (double)hi);
}

}  // namespace

struct hb_lattice {
    double kinetic, rest;
    double gamma0, bg0;
    std::vector<Elem> elems;
    std::vector<SurHost> surs;
    int run_mode = HB_RUN_COMPOSED;
    bool finalized = false;
    int device = -1;
    int sm_count = 0;
    int n_monitors = 0;
    double bg_out = 0.0;
    std::vector<Segment> segs;
    // device allocations
    HbSeqElem* d_seq = nullptr;
    double* d_partials = nullptr;
    std::vector<void*> d_bufs;
    double centroid_in[6] = {0, 0, 0, 0, 0, 0};   // nominal centroid of the incoming bunch (hb_lattice_set_centroid)
    std::vector<HbPivot> mon_pivot;               // [monitor] pivot of that record's sums
    bool timing = false;
    bool timing_valid = false;
    std::vector<cudaEvent_t> events;   // segs.size() + 1 when timing is on
    // hb_push_host: staging owned by the library, allocated at the first call and kept
    size_t host_chunk_cap = 0;         // particles per staging slot
    float* d_stage[3] = {nullptr, nullptr, nullptr};   // three staging slots: copy-in / compute / copy-out in flight
    double* d_host_partials = nullptr; // n_monitors partial buffers (one row range per chunk)
    double* d_host_records = nullptr;  // n_monitors x 27
    cudaStream_t host_streams[3] = {nullptr, nullptr, nullptr};   // copy-in, compute, copy-out
    cudaEvent_t host_events[9] = {};   // per slot: copied in, computed, copied out
    // hb_push_candidates: candidate maps and the input record (allocated at the first call, grown when K grows)
    double* d_cand_maps = nullptr;
    double* d_cand_rec = nullptr;
    int cand_cap = 0;
};

// Nominal centroid of the bunch behind every segment (host, fp64): the incoming centroid (default 0) through the
// linear(ised) run maps; a surrogate stage sends it to its output mean (R8), converted to s-coordinates about the new
// reference for COORD_T (R6, R7).  Only the conditioning of the moment sums depends on it, never their value.
static void track_pivots(hb_lattice* lat) {
    double c[6];
    for (int j = 0; j < 6; ++j) c[j] = lat->centroid_in[j];
    lat->mon_pivot.assign((size_t)lat->n_monitors, HbPivot{});
    for (Segment& g : lat->segs) {
        if (g.type == SEG_RUN) {
            double o[6];
            for (int r = 0; r < 6; ++r) {
                o[r] = 0.0;
                for (int k = 0; k < 6; ++k) o[r] += (double)g.map.m[r * 6 + k] * c[k];
            }
            for (int j = 0; j < 6; ++j) c[j] = o[j];
        } else if (g.type == SEG_SUR) {
            const SurHost& s = lat->surs[(size_t)g.sur];
            if (s.coord == HB_COORD_S) {
                for (int j = 0; j < 6; ++j) c[j] = s.out_mean[j];
            } else {
                const double ux = s.out_mean[3], uy = s.out_mean[4], uz = s.out_mean[5], z = s.out_mean[2] - g.z1;
                const double gam = std::sqrt(1.0 + ux * ux + uy * uy + uz * uz), g1 = std::sqrt(1.0 + g.bg1 * g.bg1);
                if (uz > 0.0) {
                    c[0] = s.out_mean[0] - ux / uz * z; c[1] = ux / g.bg1;
                    c[2] = s.out_mean[1] - uy / uz * z; c[3] = uy / g.bg1;
                    c[4] = -z * gam / uz;               c[5] = -(gam - g1) / g.bg1;
                } else {
                    for (int j = 0; j < 6; ++j) c[j] = 0.0;
                }
            }
            for (int j = 0; j < 6; ++j)
                if (!std::isfinite(c[j])) c[j] = 0.0;
            for (int j = 0; j < 6; ++j) g.sd.mom_pivot.p[j] = c[j];
        }
        for (int j = 0; j < 6; ++j) g.pivot[j] = c[j];
        if (g.monitor >= 0)
            for (int j = 0; j < 6; ++j) lat->mon_pivot[(size_t)g.monitor].p[j] = c[j];
    }
}

void hb_internal_set_error(const char* msg) { g_err = msg ? msg : ""; }

extern "C" {

const char* hb_status_string(hb_status s) {
    switch (s) {
    case HB_OK: return "HB_OK";
    case HB_ERR_INVALID_ARG: return "HB_ERR_INVALID_ARG";
    case HB_ERR_STATE: return "HB_ERR_STATE";
    case HB_ERR_ALLOC: return "HB_ERR_ALLOC";
    case HB_ERR_CUDA: return "HB_ERR_CUDA";
    case HB_ERR_UNSUPPORTED: return "HB_ERR_UNSUPPORTED";
    }
    return "HB_ERR_UNKNOWN";
}

const char* hb_last_error(void) { return g_err.c_str(); }

const char* hb_version(void) { return "hb 0.1 (sm_100a)"; }

const char* hb_surrogate_kernel(hb_prec prec, int n_linear, const int* widths) {
    if (!widths || n_linear < 1 || n_linear > HB_MAX_LINEAR) { fail(HB_ERR_INVALID_ARG, "n_linear / widths"); return nullptr; }
    if (widths[0] != 6 || widths[n_linear] != 6) { fail(HB_ERR_INVALID_ARG, "widths[0] and widths[last] must be 6"); return nullptr; }
    for (int l = 1; l < n_linear; ++l)
        if (widths[l] < 1 || widths[l] > HB_MAX_WIDTH) { fail(HB_ERR_INVALID_ARG, "hidden width out of range"); return nullptr; }
    if (prec == HB_PREC_FP32) return "fp32-ffma";
    char why[256];
    if (!hb_tc_supported((int)prec, n_linear, widths, why, sizeof why)) { fail(HB_ERR_UNSUPPORTED, "tensor-core surrogate: %s", why); return nullptr; }
    const int kind = hb_tc_kernel_kind((int)prec, n_linear, widths);
    return kind == 3 ? "tcgen05-layered" : (kind == 2 ? "tcgen05-streamed" : "tcgen05-resident");   // kinds 1 and 4 keep their weights in shared memory
}

hb_status hb_lattice_create(double kin, double rest, hb_lattice** out) {
    if (!out) return fail(HB_ERR_INVALID_ARG, "out is NULL");
    *out = nullptr;
    if (!std::isfinite(kin) || !std::isfinite(rest) || kin <= 0.0 || rest <= 0.0)
        return fail(HB_ERR_INVALID_ARG, "energies must be finite and positive");
    hb_lattice* l = new (std::nothrow) hb_lattice();
    if (!l) return fail(HB_ERR_ALLOC, "out of host memory");
    l->kinetic = kin;
    l->rest = rest;
    l->gamma0 = 1.0 + kin / rest;                         // R1
    l->bg0 = std::sqrt(l->gamma0 * l->gamma0 - 1.0);
    *out = l;
    return HB_OK;
}

hb_status hb_lattice_add_element(hb_lattice* lat, hb_elem_kind kind, double L, double param) {
    if (!lat) return fail(HB_ERR_INVALID_ARG, "lattice is NULL");
    if (lat->finalized) return fail(HB_ERR_STATE, "lattice already finalized");
    if (kind == HB_ELEM_MULTIPOLE) return fail(HB_ERR_INVALID_ARG, "use hb_lattice_add_multipole for a multipole kick");
    if (((int)kind < 0 || (int)kind > HB_ELEM_MONITOR) && kind != HB_ELEM_PLENS && kind != HB_ELEM_DRIFT_EXACT &&
        kind != HB_ELEM_QUAD_CHROMATIC)
        return fail(HB_ERR_INVALID_ARG, "unknown element kind %d", (int)kind);
    Elem e{(int)kind, 0.0, 0.0, -1};
    if (kind != HB_ELEM_MONITOR) {
        if (!std::isfinite(L)) return fail(HB_ERR_INVALID_ARG, "length must be finite");
        if (kind != HB_ELEM_DRIFT && kind != HB_ELEM_DRIFT_EXACT && (!std::isfinite(param) || L < 0.0))
            return fail(HB_ERR_INVALID_ARG, "quad/plens/sbend need a finite parameter and length >= 0");
        if (kind == HB_ELEM_SBEND && L == 0.0 && param != 0.0)
            return fail(HB_ERR_INVALID_ARG, "sbend of length 0 with a non-zero angle has no finite curvature (use a multipole of order 1 for a thin dipole kick)");
        e.L = L;
        e.param = (kind == HB_ELEM_DRIFT || kind == HB_ELEM_DRIFT_EXACT) ? 0.0 : param;
    }
    lat->elems.push_back(e);
    return HB_OK;
}

hb_status hb_lattice_set_element(hb_lattice* lat, int index, double L, double param) {
    if (!lat) return fail(HB_ERR_INVALID_ARG, "lattice is NULL");
    if (index < 0 || (size_t)index >= lat->elems.size())
        return fail(HB_ERR_INVALID_ARG, "element index %d out of range (lattice has %zu elements)", index, lat->elems.size());
    Elem& e = lat->elems[(size_t)index];
    if (e.kind == HB_ELEM_MONITOR || e.kind == 4 || e.kind == HB_ELEM_MULTIPOLE)
        return fail(HB_ERR_INVALID_ARG, "element %d is a monitor, surrogate or multipole: only elements added with "
                                        "hb_lattice_add_element(length, param) can be re-set", index);
    const bool is_drift = e.kind == HB_ELEM_DRIFT || e.kind == HB_ELEM_DRIFT_EXACT;
    if (!std::isfinite(L)) return fail(HB_ERR_INVALID_ARG, "length must be finite");
    if (!is_drift && (!std::isfinite(param) || L < 0.0))
        return fail(HB_ERR_INVALID_ARG, "quad/plens/sbend need a finite parameter and length >= 0");
    if (e.kind == HB_ELEM_SBEND && L == 0.0 && param != 0.0)
        return fail(HB_ERR_INVALID_ARG, "sbend of length 0 with a non-zero angle has no finite curvature");
    if (!lat->finalized) {
        e.L = L;
        e.param = is_drift ? 0.0 : param;
        return HB_OK;
    }
    // finalized: rebuild the one run that holds the element (its reference energy is fixed by the stages before it)
    for (Segment& sg : lat->segs) {
        if (sg.type != SEG_RUN || index < sg.e_lo || index >= sg.e_hi) continue;
        const Elem old = e;
        e.L = L;
        e.param = is_drift ? 0.0 : param;
        Mat6 M = mat_identity();
        std::vector<HbSeqElem> seq;
        for (int k = sg.e_lo; k < sg.e_hi; ++k) {
            M = mat_mul(elem_matrix(lat->elems[(size_t)k], sg.bg), M);
            seq.push_back(seq_elem(lat->elems[(size_t)k], sg.bg));
        }
        // the element table of sequential runs lives on the device: no push may still be reading it
        int prev = 0;
        cudaError_t ce = cudaGetDevice(&prev);
        if (ce == cudaSuccess) ce = cudaSetDevice(lat->device);
        if (ce == cudaSuccess) ce = cudaDeviceSynchronize();
        if (ce == cudaSuccess)
            ce = cudaMemcpy(lat->d_seq + sg.seq_off, seq.data(), seq.size() * sizeof(HbSeqElem), cudaMemcpyHostToDevice);
        cudaSetDevice(prev);
        if (ce != cudaSuccess) {
            e = old;
            return fail(HB_ERR_CUDA, "hb_lattice_set_element: %s", cudaGetErrorString(ce));
        }
        for (int r = 0; r < 6; ++r)
            for (int c = 0; c < 6; ++c) sg.map.m[r * 6 + c] = (float)M.m[r][c];
        track_pivots(lat);
        return HB_OK;
    }
    return fail(HB_ERR_STATE, "element %d belongs to no run", index);
}

hb_status hb_lattice_add_multipole(hb_lattice* lat, int order, double kn, double ks) {
    if (!lat) return fail(HB_ERR_INVALID_ARG, "lattice is NULL");
    if (lat->finalized) return fail(HB_ERR_STATE, "lattice already finalized");
    if (order < 1 || order > 8) return fail(HB_ERR_INVALID_ARG, "multipole order must be 1..8");
    if (!std::isfinite(kn) || !std::isfinite(ks)) return fail(HB_ERR_INVALID_ARG, "multipole strengths must be finite");
    Elem e{(int)HB_ELEM_MULTIPOLE, (double)order, kn, -1};
    e.p2 = ks;
    lat->elems.push_back(e);
    return HB_OK;
}

hb_status hb_lattice_add_surrogate(hb_lattice* lat, const hb_surrogate_desc* d) {
    if (!lat || !d) return fail(HB_ERR_INVALID_ARG, "NULL argument");
    if (lat->finalized) return fail(HB_ERR_STATE, "lattice already finalized");
    if (d->n_linear < 1 || d->n_linear > HB_MAX_LINEAR) return fail(HB_ERR_INVALID_ARG, "n_linear must be in [1,%d]", HB_MAX_LINEAR);
    if (!d->widths || !d->W || !d->b) return fail(HB_ERR_INVALID_ARG, "widths/W/b is NULL");
    if (d->widths[0] != 6 || d->widths[d->n_linear] != 6) return fail(HB_ERR_INVALID_ARG, "first and last width must be 6 (n = m = 6, P:105)");
    if ((int)d->act < 0 || (int)d->act > HB_ACT_TANH) return fail(HB_ERR_INVALID_ARG, "unknown activation");
    if ((int)d->prec < 0 || (int)d->prec > HB_PREC_TF32) return fail(HB_ERR_INVALID_ARG, "unknown precision");
    if ((int)d->coord < 0 || (int)d->coord > HB_COORD_T) return fail(HB_ERR_INVALID_ARG, "unknown coord");
    if (d->act == HB_ACT_PRELU && d->n_linear > 1 && !d->prelu_a) return fail(HB_ERR_INVALID_ARG, "PReLU needs slopes");
    SurHost s;
    s.n_linear = d->n_linear;
    s.widths.assign(d->widths, d->widths + d->n_linear + 1);
    for (int l = 1; l < d->n_linear; ++l)
        if (s.widths[l] < 1 || s.widths[l] > HB_MAX_WIDTH) return fail(HB_ERR_INVALID_ARG, "hidden width %d outside [1,%d]", s.widths[l], HB_MAX_WIDTH);
    for (int l = 0; l < d->n_linear; ++l) {
        if (!d->W[l] || !d->b[l]) return fail(HB_ERR_INVALID_ARG, "W[%d] or b[%d] is NULL", l, l);
        const size_t nw = (size_t)s.widths[l] * s.widths[l + 1];
        s.W.emplace_back(d->W[l], d->W[l] + nw);
        s.b.emplace_back(d->b[l], d->b[l] + s.widths[l + 1]);
        for (float v : s.W.back()) if (!std::isfinite(v)) return fail(HB_ERR_INVALID_ARG, "non-finite weight in layer %d", l);
        for (float v : s.b.back()) if (!std::isfinite(v)) return fail(HB_ERR_INVALID_ARG, "non-finite bias in layer %d", l);
    }
    s.act = d->act;
    s.prelu.assign(HB_MAX_LINEAR, 0.0f);
    if (d->act == HB_ACT_PRELU)
        for (int l = 0; l < d->n_linear - 1; ++l) {
            if (!std::isfinite(d->prelu_a[l])) return fail(HB_ERR_INVALID_ARG, "non-finite PReLU slope");
            s.prelu[l] = d->prelu_a[l];
        }
    for (int j = 0; j < 6; ++j) {
        if (!std::isfinite(d->in_mean[j]) || !std::isfinite(d->out_mean[j]) || !(d->in_std[j] > 0.0) ||
            !(d->out_std[j] > 0.0) || !std::isfinite(d->in_std[j]) || !std::isfinite(d->out_std[j]))
            return fail(HB_ERR_INVALID_ARG, "normalisation constants must be finite with std > 0");
        s.in_mean[j] = d->in_mean[j]; s.in_std[j] = d->in_std[j];
        s.out_mean[j] = d->out_mean[j]; s.out_std[j] = d->out_std[j];
    }
    s.coord = d->coord;
    s.ref_bg_out = d->ref_bg_out;
    s.ref_z_out = d->ref_z_out;
    if (d->coord == HB_COORD_T && !std::isnan(d->ref_bg_out) && !(d->ref_bg_out > 0.0))
        return fail(HB_ERR_INVALID_ARG, "ref_bg_out must be positive or NaN");
    s.prec = d->prec;
    lat->surs.push_back(std::move(s));
    lat->elems.push_back(Elem{4, 0.0, 0.0, (int)lat->surs.size() - 1});
    return HB_OK;
}

hb_status hb_lattice_set_run_mode(hb_lattice* lat, hb_run_mode mode) {
    if (!lat) return fail(HB_ERR_INVALID_ARG, "lattice is NULL");
    if (lat->finalized) return fail(HB_ERR_STATE, "lattice already finalized");
    if ((int)mode < 0 || (int)mode > HB_RUN_SEQUENTIAL_FP32) return fail(HB_ERR_INVALID_ARG, "unknown run mode");
    lat->run_mode = mode;
    return HB_OK;
}

hb_status hb_lattice_set_centroid(hb_lattice* lat, const double* centroid6) {
    if (!lat || !centroid6) return fail(HB_ERR_INVALID_ARG, "NULL argument");
    for (int j = 0; j < 6; ++j)
        if (!std::isfinite(centroid6[j])) return fail(HB_ERR_INVALID_ARG, "centroid must be finite");
    for (int j = 0; j < 6; ++j) lat->centroid_in[j] = centroid6[j];
    if (lat->finalized) track_pivots(lat);     // host arithmetic only; pushes enqueued earlier keep their pivots
    return HB_OK;
}

static hb_status upload(hb_lattice* lat, const void* src, size_t bytes, void** dst) {
    *dst = nullptr;
    if (bytes == 0) bytes = 16;
    void* d = nullptr;
    cudaError_t e = cudaMalloc(&d, bytes);
    if (e != cudaSuccess) return fail(HB_ERR_ALLOC, "cudaMalloc(%zu): %s", bytes, cudaGetErrorString(e));
    lat->d_bufs.push_back(d);
    if (src) HB_CUDA(cudaMemcpy(d, src, bytes, cudaMemcpyHostToDevice));
    *dst = d;
    return HB_OK;
}

static hb_status build_surrogate(hb_lattice* lat, const SurHost& s, double bg_in, double* bg_out, Segment& seg) {
    HbSurDev& sd = seg.sd;
    std::memset(&sd, 0, sizeof sd);
    sd.n_linear = s.n_linear;
    sd.act = s.act;
    sd.coord = s.coord;
    sd.prec = s.prec;
    for (int l = 0; l <= s.n_linear; ++l) sd.widths[l] = s.widths[l];
    for (int l = 0; l < HB_MAX_LINEAR; ++l) sd.prelu[l] = s.prelu[l];
    for (int j = 0; j < 6; ++j) {
        split_hi_lo(s.in_mean[j], sd.mu_hi[j], sd.mu_lo[j]);
        sd.inv_sd[j] = (float)(1.0 / s.in_std[j]);
        sd.out_sd[j] = (float)s.out_std[j];
        sd.out_mu[j] = (float)s.out_mean[j];
    }
    *bg_out = bg_in;
    if (s.coord == HB_COORD_T) {      // R6, R7
        double bg1 = s.ref_bg_out, z1 = s.ref_z_out;
        if (std::isnan(bg1) || std::isnan(z1)) {
            const double rin[6] = {0, 0, 0, 0, 0, bg_in};
            double rout[6];
            mlp_host(s, rin, rout);
            if (std::isnan(bg1)) bg1 = rout[5];
            if (std::isnan(z1)) z1 = rout[2];
        }
        if (!(bg1 > 0.0) || !std::isfinite(bg1) || !std::isfinite(z1))
            return fail(HB_ERR_INVALID_ARG, "surrogate reference output is unphysical (bg=%g, z=%g)", bg1, z1);
        const double g0 = std::sqrt(1.0 + bg_in * bg_in), g1 = std::sqrt(1.0 + bg1 * bg1);
        sd.bg0 = (float)bg_in; sd.g0 = (float)g0;
        sd.bg1 = (float)bg1; sd.g1 = (float)g1; sd.inv_bg1 = (float)(1.0 / bg1);
        sd.uz_in_shift = (float)(bg_in - s.in_mean[5]);
        sd.uz_out_shift = (float)(s.out_mean[5] - bg1);
        sd.z_out_mu = (float)(s.out_mean[2] - z1);
        seg.bg1 = bg1;
        seg.z1 = z1;
        *bg_out = bg1;
    }
    // ---- fp32 image: W^T [k][npad], zero padded to 64 outputs
    if (s.prec == HB_PREC_FP32) {
        std::vector<float> w, b;
        for (int l = 0; l < s.n_linear; ++l) {
            const int fin = s.widths[l], fout = s.widths[l + 1];
            const int npad = (fout + 63) / 64 * 64;
            sd.npad32[l] = npad;
            sd.w32_off[l] = (long long)w.size();
            sd.b32_off[l] = (int)b.size();
            w.resize(w.size() + (size_t)fin * npad, 0.0f);
            b.resize(b.size() + npad, 0.0f);
            float* wp = w.data() + sd.w32_off[l];
            for (int o = 0; o < fout; ++o)
                for (int k = 0; k < fin; ++k) wp[(size_t)k * npad + o] = s.W[l][(size_t)o * fin + k];
            for (int o = 0; o < fout; ++o) b[sd.b32_off[l] + o] = s.b[l][o];
        }
        void *dw, *db;
        hb_status st = upload(lat, w.data(), w.size() * sizeof(float), &dw);
        if (st != HB_OK) return st;
        st = upload(lat, b.data(), b.size() * sizeof(float), &db);
        if (st != HB_OK) return st;
        sd.w32 = (const float*)dw;
        sd.b32 = (const float*)db;
        sd.fp32_tp = hb_fp32_env_tp();
        seg.tc = false;
    } else {
        char why[256];
        if (!hb_tc_supported(s.prec, s.n_linear, s.widths.data(), why, sizeof why))
            return fail(HB_ERR_UNSUPPORTED, "tensor-core surrogate: %s", why);
        std::vector<const float*> Wp;
        for (int l = 0; l < s.n_linear; ++l) Wp.push_back(s.W[l].data());
        std::vector<const float*> Bp;
        for (int l = 0; l < s.n_linear; ++l) Bp.push_back(s.b[l].data());
        // kernel and launch shape are chosen here, once (test hooks of the environment included), and kept in the segment
        const HbTcChoice ch = hb_tc_choose(s.prec, s.n_linear, s.widths.data());
        sd.tc_kind = ch.kind; sd.tc_cg = ch.cg; sd.tc_g = ch.g; sd.tc_occ = ch.occ;
        const size_t bytes = hb_tc_pack_weights(ch, s.prec, s.n_linear, s.widths.data(), Wp.data(), nullptr, nullptr,
                                                sd.wtc_off, sd.kpad, sd.npadtc);
        std::vector<unsigned char> img(bytes);
        hb_tc_pack_weights(ch, s.prec, s.n_linear, s.widths.data(), Wp.data(), Bp.data(), img.data(), sd.wtc_off, sd.kpad,
                           sd.npadtc);
        std::vector<float> b;
        for (int l = 0; l < s.n_linear; ++l) {
            sd.btc_off[l] = (int)b.size();
            b.resize(b.size() + sd.npadtc[l], 0.0f);
            for (int o = 0; o < s.widths[l + 1]; ++o) b[sd.btc_off[l] + o] = s.b[l][o];
        }
        void *dw, *db;
        hb_status st = upload(lat, img.data(), img.size(), &dw);
        if (st != HB_OK) return st;
        st = upload(lat, b.data(), b.size() * sizeof(float), &db);
        if (st != HB_OK) return st;
        sd.wtc = dw;
        sd.btc = (const float*)db;
        if (sd.tc_kind == 3) {      // wide net: activations of a chunk round-trip through global scratch
            void* da = nullptr;
            st = upload(lat, nullptr, hb_tcw_scratch_bytes(s.n_linear, s.widths.data()), &da);
            if (st != HB_OK) return st;
            sd.act_scratch = (unsigned char*)da;
        }
        seg.tc = true;
    }
    // launch attributes of the kernel instantiations this stage uses (with and without fused moments): set once here
    {
        HbParticles none{};
        for (int mom = 0; mom < 2; ++mom) {
            double* fake = mom ? reinterpret_cast<double*>(sizeof(double)) : nullptr;    // only tested against nullptr
            cudaError_t e;
            if (seg.tc && sd.tc_kind == 3) e = hb_launch_sur_tcw(none, 1, sd, fake, false, nullptr, lat->sm_count, true, nullptr);
            else if (seg.tc) e = hb_launch_sur_tc(none, 1, sd, fake, nullptr, lat->sm_count, true, nullptr);
            else e = hb_launch_sur_fp32(none, 1, sd, fake, nullptr, lat->sm_count, true, nullptr);
            if (e != cudaSuccess) return fail(HB_ERR_CUDA, "surrogate kernel attributes: %s", cudaGetErrorString(e));
        }
    }
    return HB_OK;
}

hb_status hb_lattice_finalize(hb_lattice* lat, int device) {
    if (!lat) return fail(HB_ERR_INVALID_ARG, "lattice is NULL");
    if (lat->finalized) return fail(HB_ERR_STATE, "lattice already finalized");
    int ndev = 0;
    HB_CUDA(cudaGetDeviceCount(&ndev));
    if (device < 0 || device >= ndev) return fail(HB_ERR_CUDA, "no CUDA device %d (have %d)", device, ndev);
    cudaDeviceProp prop;
    HB_CUDA(cudaGetDeviceProperties(&prop, device));
    if (prop.major != 10 || prop.minor != 0)
        return fail(HB_ERR_UNSUPPORTED, "device %d is sm_%d%d; libhb is built for sm_100a only", device, prop.major, prop.minor);
    if (prop.multiProcessorCount * 4 > HB_MOM_GRID_MAX)
        return fail(HB_ERR_UNSUPPORTED, "device %d has %d SMs; the moment-partials layout is sized for <= %d", device,
                    prop.multiProcessorCount, HB_MOM_GRID_MAX / 4);
    int prev = 0;
    HB_CUDA(cudaGetDevice(&prev));
    HB_CUDA(cudaSetDevice(device));
    lat->device = device;
    lat->sm_count = prop.multiProcessorCount;

    // ---- split into segments, tracking the reference (R5, R7, G17)
    std::vector<HbSeqElem> seq;
    double bg = lat->bg0;
    lat->segs.clear();
    lat->n_monitors = 0;
    size_t i = 0;
    hb_status st = HB_OK;
    while (i < lat->elems.size() && st == HB_OK) {
        const Elem& e = lat->elems[i];
        if (e.kind == HB_ELEM_MONITOR) {
            if (!lat->segs.empty() && lat->segs.back().monitor < 0 && lat->segs.back().type != SEG_MON) {
                lat->segs.back().monitor = lat->n_monitors++;
            } else {
                Segment s{};
                s.type = SEG_MON;
                s.monitor = lat->n_monitors++;
                lat->segs.push_back(s);
            }
            ++i;
        } else if (e.kind == 4) {
            Segment s{};
            s.type = SEG_SUR;
            s.monitor = -1;
            s.sur = e.sur;
            double bg1 = bg;
            st = build_surrogate(lat, lat->surs[e.sur], bg, &bg1, s);
            bg = bg1;
            lat->segs.push_back(s);
            ++i;
        } else {
            Segment s{};
            s.type = SEG_RUN;
            s.monitor = -1;
            s.seq_off = (int)seq.size();
            s.e_lo = (int)i;
            s.bg = bg;
            Mat6 M = mat_identity();
            while (i < lat->elems.size() && is_conventional(lat->elems[i].kind)) {
                s.nonlinear = s.nonlinear || is_nonlinear(lat->elems[i].kind);
                M = mat_mul(elem_matrix(lat->elems[i], bg), M);
                seq.push_back(seq_elem(lat->elems[i], bg));
                ++i;
            }
            s.seq_cnt = (int)seq.size() - s.seq_off;
            s.e_hi = (int)i;
            for (int r = 0; r < 6; ++r)
                for (int c = 0; c < 6; ++c) s.map.m[r * 6 + c] = (float)M.m[r][c];
            lat->segs.push_back(s);
        }
    }
    if (st == HB_OK) {
        void* d = nullptr;
        st = upload(lat, seq.data(), seq.size() * sizeof(HbSeqElem), &d);
        lat->d_seq = (HbSeqElem*)d;
    }
    if (st == HB_OK) {
        void* d = nullptr;
        st = upload(lat, nullptr, (size_t)HB_MOM_MAX_BLOCKS * HB_NMOM * sizeof(double), &d);
        lat->d_partials = (double*)d;
    }
    if (st == HB_OK) {
        cudaError_t e = cudaDeviceSynchronize();
        if (e != cudaSuccess) st = fail(HB_ERR_CUDA, "cudaDeviceSynchronize: %s", cudaGetErrorString(e));
    }
    lat->bg_out = bg;
    if (st == HB_OK) track_pivots(lat);
    cudaSetDevice(prev);
    if (st != HB_OK) {
        for (void* p : lat->d_bufs) cudaFree(p);
        lat->d_bufs.clear();
        lat->segs.clear();
        return st;
    }
    lat->finalized = true;
    return HB_OK;
}

hb_status hb_lattice_num_monitors(const hb_lattice* lat, int* out) {
    if (!lat || !out) return fail(HB_ERR_INVALID_ARG, "NULL argument");
    int n = 0;
    for (const Elem& e : lat->elems) n += e.kind == HB_ELEM_MONITOR;
    *out = n;
    return HB_OK;
}

hb_status hb_lattice_num_launches(const hb_lattice* lat, int with_moments, size_t n_particles, int* out) {
    if (!lat || !out) return fail(HB_ERR_INVALID_ARG, "NULL argument");
    if (!lat->finalized) return fail(HB_ERR_STATE, "lattice not finalized");
    int n = 0;
    if (n_particles > 0)
        for (const Segment& s : lat->segs) {
            if (s.type == SEG_MON) { n += with_moments ? 2 : 0; continue; }
            // a layered (wide-net) stage is one launch per linear layer and chunk of HB_TCW_CHUNK particles
            if (s.type == SEG_SUR && s.tc && s.sd.tc_kind == 3)
                n += (int)((n_particles + HB_TCW_CHUNK - 1) / HB_TCW_CHUNK) * s.sd.n_linear;
            else n += 1;
            n += (with_moments && s.monitor >= 0) ? 1 : 0;
        }
    *out = n;
    return HB_OK;
}

hb_status hb_lattice_ref_bg_out(const hb_lattice* lat, double* out) {
    if (!lat || !out) return fail(HB_ERR_INVALID_ARG, "NULL argument");
    if (!lat->finalized) return fail(HB_ERR_STATE, "lattice not finalized");
    *out = lat->bg_out;
    return HB_OK;
}

static hb_status check_arrays(const float* const a[6], size_t n) {
    for (int j = 0; j < 6; ++j) {
        if (!a[j]) return fail(HB_ERR_INVALID_ARG, "particle array %d is NULL", j);
        if ((uintptr_t)a[j] & 15u) return fail(HB_ERR_INVALID_ARG, "particle array %d is not 16-byte aligned", j);
    }
    const size_t bytes = n * sizeof(float);
    for (int j = 0; j < 6; ++j)
        for (int k = j + 1; k < 6; ++k) {
            const uintptr_t a0 = (uintptr_t)a[j], b0 = (uintptr_t)a[k];
            if (a0 < b0 + bytes && b0 < a0 + bytes)
                return fail(HB_ERR_INVALID_ARG, "particle arrays %d and %d overlap", j, k);
        }
    return HB_OK;
}

// Enqueue every segment of the lattice for the particles p[0..n) on stream s.
//   host_partials == nullptr : moment partials go to lat->d_partials and each record is finalized at once into d_moments
//   host_partials != nullptr : (hb_push_host, one call per chunk) the partials of monitor m go to rows
//                              [row_off, row_off + blocks) of host_partials + m * 27 * HB_MOM_MAX_BLOCKS; no finalize
static hb_status enqueue_segments(hb_lattice* lat, const HbParticles& p, size_t n, bool want_moments, double* d_moments,
                                  double* host_partials, size_t row_off, bool timing, cudaStream_t s) {
    hb_status st = HB_OK;
    for (size_t k = 0; k < lat->segs.size() && st == HB_OK; ++k) {
        const Segment& g = lat->segs[k];
        const bool mom = want_moments && g.monitor >= 0;
        double* partials = nullptr;
        if (mom) partials = host_partials ? host_partials + (size_t)g.monitor * HB_NMOM * HB_MOM_MAX_BLOCKS + row_off : lat->d_partials;
        int nblocks = 0;
        cudaError_t e = cudaSuccess;
        if (g.type == SEG_RUN) {
            if (lat->run_mode == HB_RUN_COMPOSED && !g.nonlinear) e = hb_launch_run_composed(p, n, g.map, g.pivot, partials, &nblocks, s);
            else e = hb_launch_run_sequential(p, n, lat->d_seq + g.seq_off, g.seq_cnt,
                                              lat->run_mode == HB_RUN_SEQUENTIAL_FP32, g.nonlinear, g.pivot, partials, &nblocks, s);
        } else if (g.type == SEG_SUR) {
            if (g.tc && g.sd.tc_kind == 3) e = hb_launch_sur_tcw(p, n, g.sd, partials, host_partials != nullptr, &nblocks, lat->sm_count, false, s);
            else e = g.tc ? hb_launch_sur_tc(p, n, g.sd, partials, &nblocks, lat->sm_count, false, s)
                          : hb_launch_sur_fp32(p, n, g.sd, partials, &nblocks, lat->sm_count, false, s);
        } else if (mom) {
            e = hb_launch_moments_partials(p, n, g.pivot, partials, &nblocks, s);
        }
        if (e != cudaSuccess) { st = fail(HB_ERR_CUDA, "kernel launch (segment %zu): %s", k, cudaGetErrorString(e)); break; }
        if (mom && !host_partials) {
            e = hb_launch_moments_finalize(partials, nblocks, n, g.pivot, d_moments + (size_t)g.monitor * HB_NMOM, s);
            if (e != cudaSuccess) st = fail(HB_ERR_CUDA, "moments finalize: %s", cudaGetErrorString(e));
        }
        if (timing) cudaEventRecord(lat->events[k + 1], s);
    }
    return st;
}

static hb_status push_impl(hb_lattice* lat, float* x, float* px, float* y, float* py, float* t, float* pt, size_t n,
                           double* d_moments, bool want_moments, void* stream) {
    if (!lat) return fail(HB_ERR_INVALID_ARG, "lattice is NULL");
    if (!lat->finalized) return fail(HB_ERR_STATE, "lattice not finalized");
    cudaStream_t s = (cudaStream_t)stream;
    if (want_moments && lat->n_monitors > 0) {
        if (!d_moments) return fail(HB_ERR_INVALID_ARG, "d_moments is NULL");
        if ((uintptr_t)d_moments & 7u) return fail(HB_ERR_INVALID_ARG, "d_moments is not 8-byte aligned");
    }
    int prev = 0;
    HB_CUDA(cudaGetDevice(&prev));
    if (prev != lat->device) HB_CUDA(cudaSetDevice(lat->device));
    hb_status st = HB_OK;
    if (n == 0) {
        if (want_moments && lat->n_monitors > 0) {    // NaN records: all-ones bytes are a quiet NaN
            cudaError_t e = cudaMemsetAsync(d_moments, 0xff, (size_t)lat->n_monitors * HB_NMOM * sizeof(double), s);
            if (e != cudaSuccess) st = fail(HB_ERR_CUDA, "cudaMemsetAsync: %s", cudaGetErrorString(e));
        }
    } else {
        const float* arr[6] = {x, px, y, py, t, pt};
        st = check_arrays(arr, n);
        HbParticles p;
        p.v[0] = x; p.v[1] = px; p.v[2] = y; p.v[3] = py; p.v[4] = t; p.v[5] = pt;
        const bool timing = lat->timing && lat->events.size() == lat->segs.size() + 1;
        lat->timing_valid = false;
        if (timing) cudaEventRecord(lat->events[0], s);
        if (st == HB_OK) st = enqueue_segments(lat, p, n, want_moments, d_moments, nullptr, 0, timing, s);
        if (timing && st == HB_OK) lat->timing_valid = true;
    }
    if (prev != lat->device) cudaSetDevice(prev);
    return st;
}

hb_status hb_push(hb_lattice* lat, float* x, float* px, float* y, float* py, float* t, float* pt, size_t n, void* stream) {
    return push_impl(lat, x, px, y, py, t, pt, n, nullptr, false, stream);
}

hb_status hb_push_moments(hb_lattice* lat, float* x, float* px, float* y, float* py, float* t, float* pt, size_t n,
                          double* d_moments, void* stream) {
    return push_impl(lat, x, px, y, py, t, pt, n, d_moments, true, stream);
}

// ---- host-resident bunch: H2D, push, D2H pipelined in chunks over two internal streams ------------------------
hb_status hb_push_host(hb_lattice* lat, float* x, float* px, float* y, float* py, float* t, float* pt, size_t n,
                       double* h_moments, int chunks) {
    if (!lat) return fail(HB_ERR_INVALID_ARG, "lattice is NULL");
    if (!lat->finalized) return fail(HB_ERR_STATE, "lattice not finalized");
    if (chunks < 1 || chunks > HB_MOM_MAX_BLOCKS / HB_MOM_GRID_MAX)
        return fail(HB_ERR_INVALID_ARG, "chunks must be 1..%d", HB_MOM_MAX_BLOCKS / HB_MOM_GRID_MAX);
    float* host[6] = {x, px, y, py, t, pt};
    if (n > 0) {
        const float* arr[6] = {x, px, y, py, t, pt};
        for (int j = 0; j < 6; ++j)
            if (!arr[j]) return fail(HB_ERR_INVALID_ARG, "particle array %d is NULL", j);
        const size_t bytes = n * sizeof(float);
        for (int j = 0; j < 6; ++j)
            for (int k = j + 1; k < 6; ++k) {
                const uintptr_t a0 = (uintptr_t)arr[j], b0 = (uintptr_t)arr[k];
                if (a0 < b0 + bytes && b0 < a0 + bytes) return fail(HB_ERR_INVALID_ARG, "particle arrays %d and %d overlap", j, k);
            }
    }
    const bool want = h_moments != nullptr && lat->n_monitors > 0;
    if (n == 0) {
        if (want) std::memset(h_moments, 0xff, (size_t)lat->n_monitors * HB_NMOM * sizeof(double));   // NaN records
        return HB_OK;
    }
    int prev = 0;
    HB_CUDA(cudaGetDevice(&prev));
    if (prev != lat->device) HB_CUDA(cudaSetDevice(lat->device));
    // particles per chunk: whole 256-particle tile pairs, 16-byte aligned device rows
    size_t chunk_n = (n + (size_t)chunks - 1) / (size_t)chunks;
    chunk_n = (chunk_n + 255) / 256 * 256;
    hb_status st = HB_OK;
    // ---- resources, once (and again if a larger chunk is asked for)
    if (!lat->host_streams[0]) {
        for (int i = 0; i < 3 && st == HB_OK; ++i)
            if (cudaStreamCreateWithFlags(&lat->host_streams[i], cudaStreamNonBlocking) != cudaSuccess)
                st = fail(HB_ERR_CUDA, "stream creation failed");
        for (int i = 0; i < 9 && st == HB_OK; ++i)
            if (cudaEventCreateWithFlags(&lat->host_events[i], cudaEventDisableTiming) != cudaSuccess)
                st = fail(HB_ERR_CUDA, "event creation failed");
        if (st == HB_OK && lat->n_monitors > 0) {
            void* d = nullptr;
            st = upload(lat, nullptr, (size_t)lat->n_monitors * HB_NMOM * HB_MOM_MAX_BLOCKS * sizeof(double), &d);
            lat->d_host_partials = (double*)d;
            if (st == HB_OK) st = upload(lat, nullptr, (size_t)lat->n_monitors * HB_NMOM * sizeof(double), &d);
            lat->d_host_records = (double*)d;
        }
    }
    if (st == HB_OK && chunk_n > lat->host_chunk_cap) {
        // outgrown staging slots are freed first (the previous hb_push_host returned only after its streams had drained)
        for (int i = 0; i < 3; ++i) {
            if (!lat->d_stage[i]) continue;
            for (size_t k = 0; k < lat->d_bufs.size(); ++k)
                if (lat->d_bufs[k] == (void*)lat->d_stage[i]) { lat->d_bufs.erase(lat->d_bufs.begin() + (long)k); break; }
            cudaFree(lat->d_stage[i]);
            lat->d_stage[i] = nullptr;
        }
        lat->host_chunk_cap = 0;
        for (int i = 0; i < 3 && st == HB_OK; ++i) {
            void* d = nullptr;
            st = upload(lat, nullptr, 6 * chunk_n * sizeof(float), &d);
            lat->d_stage[i] = (float*)d;
        }
        if (st == HB_OK) lat->host_chunk_cap = chunk_n;
    }
    if (st == HB_OK) {
        // three-stage pipeline over three staging slots: the copy engine of each direction and the SMs each work
        // on a different piece; events hand a slot from stage to stage
        cudaStream_t sin = lat->host_streams[0], scmp = lat->host_streams[1], sout = lat->host_streams[2];
        cudaEvent_t* ev_in = lat->host_events;          // [slot] piece copied in
        cudaEvent_t* ev_k = lat->host_events + 3;       // [slot] piece computed
        cudaEvent_t* ev_out = lat->host_events + 6;     // [slot] piece copied out (slot free again)
        cudaError_t e = cudaSuccess;
        if (want)        // rows a piece does not write must read as zero in the finalize
            e = cudaMemsetAsync(lat->d_host_partials, 0, (size_t)lat->n_monitors * HB_NMOM * HB_MOM_MAX_BLOCKS * sizeof(double), scmp);
        size_t off = 0;
        int pieces = 0;
        for (int c = 0; c < chunks && off < n && st == HB_OK && e == cudaSuccess; ++c, ++pieces) {
            const size_t nc = n - off < chunk_n ? n - off : chunk_n;
            const int slot = c % 3;
            float* base = lat->d_stage[slot];
            HbParticles p;
            if (c >= 3) e = cudaStreamWaitEvent(sin, ev_out[slot], 0);
            for (int j = 0; j < 6 && e == cudaSuccess; ++j) {
                p.v[j] = base + (size_t)j * lat->host_chunk_cap;
                e = cudaMemcpyAsync(p.v[j], host[j] + off, nc * sizeof(float), cudaMemcpyHostToDevice, sin);
            }
            if (e == cudaSuccess) e = cudaEventRecord(ev_in[slot], sin);
            if (e == cudaSuccess) e = cudaStreamWaitEvent(scmp, ev_in[slot], 0);
            if (e != cudaSuccess) break;
            st = enqueue_segments(lat, p, nc, want, nullptr, want ? lat->d_host_partials : nullptr,
                                  (size_t)c * HB_MOM_GRID_MAX, false, scmp);
            if (st != HB_OK) break;
            e = cudaEventRecord(ev_k[slot], scmp);
            if (e == cudaSuccess) e = cudaStreamWaitEvent(sout, ev_k[slot], 0);
            for (int j = 0; j < 6 && e == cudaSuccess; ++j)
                e = cudaMemcpyAsync(host[j] + off, p.v[j], nc * sizeof(float), cudaMemcpyDeviceToHost, sout);
            if (e == cudaSuccess) e = cudaEventRecord(ev_out[slot], sout);
            off += nc;
        }
        if (e == cudaSuccess && st == HB_OK && want) {
            for (int m = 0; m < lat->n_monitors && e == cudaSuccess; ++m)
                e = hb_launch_moments_finalize(lat->d_host_partials + (size_t)m * HB_NMOM * HB_MOM_MAX_BLOCKS,
                                               pieces * HB_MOM_GRID_MAX, n, lat->mon_pivot[(size_t)m].p,
                                               lat->d_host_records + (size_t)m * HB_NMOM, scmp);
            if (e == cudaSuccess)
                e = cudaMemcpyAsync(h_moments, lat->d_host_records, (size_t)lat->n_monitors * HB_NMOM * sizeof(double),
                                    cudaMemcpyDeviceToHost, scmp);
        }
        const cudaError_t e1 = cudaStreamSynchronize(sin), e2 = cudaStreamSynchronize(scmp), e3 = cudaStreamSynchronize(sout);
        if (e == cudaSuccess) e = e1 != cudaSuccess ? e1 : (e2 != cudaSuccess ? e2 : e3);
        if (e != cudaSuccess && st == HB_OK) st = fail(HB_ERR_CUDA, "hb_push_host: %s", cudaGetErrorString(e));
    }
    if (prev != lat->device) cudaSetDevice(prev);
    return st;
}

hb_status hb_push_candidates(hb_lattice* lat, int n_candidates, int n_set, const int* elem_index, const double* length_m,
                             const double* param, const float* x, const float* px, const float* y, const float* py,
                             const float* t, const float* pt, size_t n, double* d_moments, void* stream) {
    if (!lat) return fail(HB_ERR_INVALID_ARG, "lattice is NULL");
    if (!lat->finalized) return fail(HB_ERR_STATE, "lattice not finalized");
    if (n_candidates < 0 || n_candidates > 65536) return fail(HB_ERR_INVALID_ARG, "n_candidates must be 0..65536");
    if (n_set < 1 || n_set > 64 || !elem_index || !length_m || !param) return fail(HB_ERR_INVALID_ARG, "n_set must be 1..64 with elem_index / length_m / param given");
    if (n_candidates > 0 && !d_moments) return fail(HB_ERR_INVALID_ARG, "d_moments is NULL");
    if ((uintptr_t)d_moments & 7u) return fail(HB_ERR_INVALID_ARG, "d_moments is not 8-byte aligned");
    // the run that holds the elements: all of them in the same one, which must be linear
    const Segment* run = nullptr;
    for (const Segment& sg : lat->segs)
        if (sg.type == SEG_RUN && elem_index[0] >= sg.e_lo && elem_index[0] < sg.e_hi) run = &sg;
    if (!run) return fail(HB_ERR_INVALID_ARG, "element %d belongs to no run of conventional elements", elem_index[0]);
    if (run->nonlinear) return fail(HB_ERR_UNSUPPORTED, "the run holds a non-linear element: it has no composed map to vary");
    for (int j = 0; j < n_set; ++j) {
        const int e = elem_index[j];
        if (e < run->e_lo || e >= run->e_hi) return fail(HB_ERR_INVALID_ARG, "element %d is not in the run of element %d", e, elem_index[0]);
        if (lat->elems[(size_t)e].kind == HB_ELEM_MULTIPOLE) return fail(HB_ERR_INVALID_ARG, "element %d is a multipole", e);
    }
    cudaStream_t s = (cudaStream_t)stream;
    int prev = 0;
    HB_CUDA(cudaGetDevice(&prev));
    if (prev != lat->device) HB_CUDA(cudaSetDevice(lat->device));
    hb_status st = HB_OK;
    if (n_candidates > 0 && n == 0) {
        cudaError_t e = cudaMemsetAsync(d_moments, 0xff, (size_t)n_candidates * HB_NMOM * sizeof(double), s);   // NaN records
        if (e != cudaSuccess) st = fail(HB_ERR_CUDA, "cudaMemsetAsync: %s", cudaGetErrorString(e));
    } else if (n_candidates > 0) {
        const float* arr[6] = {x, px, y, py, t, pt};
        st = check_arrays(arr, n);
        // candidate maps: the run's elements with the listed ones re-set, concatenated in fp64 (R5), as in finalize
        std::vector<double> maps((size_t)n_candidates * 36);
        for (int k = 0; k < n_candidates && st == HB_OK; ++k) {
            Mat6 M = mat_identity();
            for (int q = run->e_lo; q < run->e_hi; ++q) {
                Elem el = lat->elems[(size_t)q];
                for (int j = 0; j < n_set; ++j)
                    if (elem_index[j] == q) {
                        const double Lk = length_m[(size_t)k * n_set + j], pk = param[(size_t)k * n_set + j];
                        const bool is_drift = el.kind == HB_ELEM_DRIFT;
                        if (!std::isfinite(Lk) || (!is_drift && (!std::isfinite(pk) || Lk < 0.0)) ||
                            (el.kind == HB_ELEM_SBEND && Lk == 0.0 && pk != 0.0)) {
                            st = fail(HB_ERR_INVALID_ARG, "candidate %d: invalid length / parameter for element %d", k, q);
                            break;
                        }
                        el.L = Lk;
                        el.param = is_drift ? 0.0 : pk;
                    }
                M = mat_mul(elem_matrix(el, run->bg), M);
            }
            for (int r = 0; r < 6; ++r)
                for (int c = 0; c < 6; ++c) maps[(size_t)k * 36 + r * 6 + c] = M.m[r][c];
        }
        if (st == HB_OK && n_candidates > lat->cand_cap) {
            // (grown buffers: the old ones stay until destroy -- a push enqueued earlier may still read them)
            void* d = nullptr;
            st = upload(lat, nullptr, (size_t)n_candidates * 36 * sizeof(double), &d);
            lat->d_cand_maps = (double*)d;
            if (st == HB_OK && !lat->d_cand_rec) {
                st = upload(lat, nullptr, HB_NMOM * sizeof(double), &d);
                lat->d_cand_rec = (double*)d;
            }
            if (st == HB_OK) lat->cand_cap = n_candidates;
        }
        if (st == HB_OK) {
            HbParticles p;
            for (int j = 0; j < 6; ++j) p.v[j] = const_cast<float*>(arr[j]);
            // pivot: the nominal centroid of the state that enters the run (= behind the segment before it)
            const double* pivot = lat->centroid_in;
            for (const Segment& sg : lat->segs) {
                if (&sg == run) break;
                pivot = sg.pivot;
            }
            int nblocks = 0;
            cudaError_t e = cudaMemcpyAsync(lat->d_cand_maps, maps.data(), maps.size() * sizeof(double), cudaMemcpyHostToDevice, s);
            if (e == cudaSuccess) e = hb_launch_moments_partials(p, n, pivot, lat->d_partials, &nblocks, s);
            if (e == cudaSuccess) e = hb_launch_moments_finalize(lat->d_partials, nblocks, n, pivot, lat->d_cand_rec, s);
            if (e == cudaSuccess) e = hb_launch_candidates(lat->d_cand_rec, lat->d_cand_maps, n_candidates, d_moments, s);
            if (e != cudaSuccess) st = fail(HB_ERR_CUDA, "hb_push_candidates: %s", cudaGetErrorString(e));
        }
    }
    if (prev != lat->device) cudaSetDevice(prev);
    return st;
}

hb_status hb_moments_merge(const double* rec_a, unsigned long long n_a, const double* rec_b, unsigned long long n_b,
                           double* rec_out) {
    if (!rec_a || !rec_b || !rec_out) return fail(HB_ERR_INVALID_ARG, "hb_moments_merge: NULL record");
    double out[HB_NMOM];
    if (n_a == 0 && n_b == 0) {
        for (int i = 0; i < HB_NMOM; ++i) out[i] = std::numeric_limits<double>::quiet_NaN();
    } else if (n_a == 0 || n_b == 0) {
        const double* src = n_a ? rec_a : rec_b;
        for (int i = 0; i < HB_NMOM; ++i) out[i] = src[i];
    } else {
        const double na = (double)n_a, nb = (double)n_b, n = na + nb;
        const double wa = na / n, wb = nb / n;
        double d[6];
        for (int i = 0; i < 6; ++i) {
            d[i] = rec_b[i] - rec_a[i];
            out[i] = rec_a[i] + wb * d[i];
        }
        int k = 6;
        for (int i = 0; i < 6; ++i)
            for (int j = i; j < 6; ++j, ++k) out[k] = wa * rec_a[k] + wb * rec_b[k] + wa * wb * d[i] * d[j];
    }
    for (int i = 0; i < HB_NMOM; ++i) rec_out[i] = out[i];
    return HB_OK;
}

size_t hb_moments_scratch_bytes(void) { return (size_t)HB_MOM_MAX_BLOCKS * HB_NMOM * sizeof(double); }

hb_status hb_moments(const float* x, const float* px, const float* y, const float* py, const float* t, const float* pt,
                     size_t n, const double* pivot, double* d_out27, void* d_scratch, void* stream) {
    if (!d_out27 || !d_scratch) return fail(HB_ERR_INVALID_ARG, "d_out27 / d_scratch is NULL");
    cudaStream_t s = (cudaStream_t)stream;
    if (n == 0) {
        HB_CUDA(cudaMemsetAsync(d_out27, 0xff, HB_NMOM * sizeof(double), s));
        return HB_OK;
    }
    const float* arr[6] = {x, px, y, py, t, pt};
    hb_status st = check_arrays(arr, n);
    if (st != HB_OK) return st;
    HbParticles p;
    for (int j = 0; j < 6; ++j) p.v[j] = const_cast<float*>(arr[j]);
    int nblocks = 0;
    HB_CUDA(hb_launch_moments_partials(p, n, pivot, (double*)d_scratch, &nblocks, s));
    HB_CUDA(hb_launch_moments_finalize((const double*)d_scratch, nblocks, n, pivot, d_out27, s));
    return HB_OK;
}

hb_status hb_lattice_enable_timing(hb_lattice* lat, int on) {
    if (!lat) return fail(HB_ERR_INVALID_ARG, "lattice is NULL");
    if (!lat->finalized) return fail(HB_ERR_STATE, "lattice not finalized");
    int prev = 0;
    HB_CUDA(cudaGetDevice(&prev));
    HB_CUDA(cudaSetDevice(lat->device));
    if (on && lat->events.empty()) {
        lat->events.resize(lat->segs.size() + 1);
        for (auto& ev : lat->events) HB_CUDA(cudaEventCreate(&ev));
    }
    lat->timing = on != 0;
    lat->timing_valid = false;
    cudaSetDevice(prev);
    return HB_OK;
}

hb_status hb_lattice_get_timing(hb_lattice* lat, float* ms_out, int capacity, int* n_out) {
    if (!lat || !n_out) return fail(HB_ERR_INVALID_ARG, "NULL argument");
    if (!lat->finalized || !lat->timing || !lat->timing_valid) return fail(HB_ERR_STATE, "no timed push to report");
    HB_CUDA(cudaEventSynchronize(lat->events.back()));
    const int n = (int)lat->segs.size();
    *n_out = n;
    for (int k = 0; k < n && k < capacity && ms_out; ++k)
        HB_CUDA(cudaEventElapsedTime(&ms_out[k], lat->events[k], lat->events[k + 1]));
    return HB_OK;
}

hb_status hb_lattice_destroy(hb_lattice* lat) {
    if (!lat) return HB_OK;
    if (lat->finalized) {
        int prev = 0;
        cudaGetDevice(&prev);
        cudaSetDevice(lat->device);
        cudaDeviceSynchronize();
        for (auto& ev : lat->events) cudaEventDestroy(ev);
        for (int i = 0; i < 9; ++i)
            if (lat->host_events[i]) cudaEventDestroy(lat->host_events[i]);
        for (int i = 0; i < 3; ++i)
            if (lat->host_streams[i]) cudaStreamDestroy(lat->host_streams[i]);
        for (void* p : lat->d_bufs) cudaFree(p);
        cudaSetDevice(prev);
    }
    delete lat;
    return HB_OK;
}

}  // extern "C"
