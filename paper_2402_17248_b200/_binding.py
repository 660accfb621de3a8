"""ctypes marshalling for include/hb.h.  Same names as the C ABI; plus `Lattice`, a small RAII wrapper."""
from __future__ import annotations

import ctypes
import math
import os
from ctypes import POINTER, c_char_p, c_double, c_float, c_int, c_size_t, c_void_p

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libhb.so")

ELEM_KINDS = {"drift": 0, "quad": 1, "sbend": 2, "monitor": 3, "plens": 5, "drift_exact": 6, "quad_chromatic": 7}
ACTS = {"identity": 0, "relu": 1, "prelu": 2, "tanh": 3}
PRECS = {"fp32": 0, "bf16": 1, "f16": 2, "tf32": 3}
COORDS = {"s": 0, "t": 1}
RUN_MODES = {"composed": 0, "sequential": 1, "sequential_fp32": 2}

EXPORTED_SYMBOLS = [
    "hb_lattice_create", "hb_lattice_add_element", "hb_lattice_set_element", "hb_lattice_add_multipole",
    "hb_lattice_add_surrogate",
    "hb_lattice_set_run_mode", "hb_lattice_set_centroid",
    "hb_lattice_finalize", "hb_lattice_num_monitors", "hb_lattice_num_launches", "hb_lattice_ref_bg_out",
    "hb_push", "hb_push_moments", "hb_push_host", "hb_push_candidates", "hb_moments", "hb_moments_scratch_bytes", "hb_moments_merge",
    "hb_moments_static", "hb_moments_static_max_particles",
    "hb_lattice_destroy",
    "hb_lattice_enable_timing", "hb_lattice_get_timing",
    "hb_status_string", "hb_last_error", "hb_version", "hb_surrogate_kernel", "hb_device_peaks",
]


class HbError(RuntimeError):
    def __init__(self, status, where):
        self.status = int(status)
        msg = "%s: %s (%s)" % (where, hb_status_string(status), hb_last_error())
        super().__init__(msg)


class _SurrogateDesc(ctypes.Structure):
    _fields_ = [
        ("n_linear", c_int),
        ("widths", POINTER(c_int)),
        ("W", POINTER(POINTER(c_float))),
        ("b", POINTER(POINTER(c_float))),
        ("act", c_int),
        ("prelu_a", POINTER(c_float)),
        ("in_mean", c_double * 6), ("in_std", c_double * 6),
        ("out_mean", c_double * 6), ("out_std", c_double * 6),
        ("coord", c_int),
        ("ref_bg_out", c_double),
        ("ref_z_out", c_double),
        ("prec", c_int),
    ]


_lib = None


def lib_path() -> str:
    return _LIB_PATH


def lib():
    """Load libhb.so (built in-tree by paper_2402_17248_b200/build.py).  Fails loudly if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise ImportError("libhb.so is not built: run `python -c 'import __graft_entry__ as g; g.build()'` "
                          "(there is no CPU fallback)")
    L = ctypes.CDLL(_LIB_PATH)
    fp = POINTER(c_float)
    L.hb_lattice_create.argtypes = [c_double, c_double, POINTER(c_void_p)]
    L.hb_lattice_add_element.argtypes = [c_void_p, c_int, c_double, c_double]
    L.hb_lattice_add_multipole.argtypes = [c_void_p, c_int, c_double, c_double]
    L.hb_lattice_set_element.argtypes = [c_void_p, c_int, c_double, c_double]
    L.hb_lattice_add_surrogate.argtypes = [c_void_p, POINTER(_SurrogateDesc)]
    L.hb_lattice_set_run_mode.argtypes = [c_void_p, c_int]
    L.hb_lattice_finalize.argtypes = [c_void_p, c_int]
    L.hb_lattice_num_monitors.argtypes = [c_void_p, POINTER(c_int)]
    L.hb_lattice_num_launches.argtypes = [c_void_p, c_int, c_size_t, POINTER(c_int)]
    L.hb_lattice_set_centroid.argtypes = [c_void_p, POINTER(c_double)]
    L.hb_lattice_ref_bg_out.argtypes = [c_void_p, POINTER(c_double)]
    L.hb_push.argtypes = [c_void_p] + [c_void_p] * 6 + [c_size_t, c_void_p]
    L.hb_push_moments.argtypes = [c_void_p] + [c_void_p] * 6 + [c_size_t, c_void_p, c_void_p]
    L.hb_push_host.argtypes = [c_void_p] + [c_void_p] * 6 + [c_size_t, c_void_p, c_int]
    L.hb_push_candidates.argtypes = [c_void_p, c_int, c_int, POINTER(c_int), POINTER(c_double), POINTER(c_double)] + \
        [c_void_p] * 6 + [c_size_t, c_void_p, c_void_p]
    L.hb_moments.argtypes = [c_void_p] * 6 + [c_size_t, POINTER(c_double), c_void_p, c_void_p, c_void_p]
    L.hb_moments_scratch_bytes.restype = c_size_t
    L.hb_moments_scratch_bytes.argtypes = []
    L.hb_moments_static.argtypes = [c_void_p] * 6 + [c_size_t, POINTER(c_double), c_void_p, c_void_p]
    L.hb_moments_static_max_particles.restype = c_size_t
    L.hb_moments_static_max_particles.argtypes = []
    L.hb_moments_merge.argtypes = [POINTER(c_double), ctypes.c_ulonglong, POINTER(c_double), ctypes.c_ulonglong,
                                   POINTER(c_double)]
    L.hb_lattice_destroy.argtypes = [c_void_p]
    L.hb_lattice_enable_timing.argtypes = [c_void_p, c_int]
    L.hb_lattice_get_timing.argtypes = [c_void_p, POINTER(c_float), c_int, POINTER(c_int)]
    L.hb_status_string.restype = c_char_p
    L.hb_status_string.argtypes = [c_int]
    L.hb_last_error.restype = c_char_p
    L.hb_version.restype = c_char_p
    L.hb_device_peaks.argtypes = [c_int, POINTER(c_double)]
    L.hb_surrogate_kernel.restype = c_char_p
    L.hb_surrogate_kernel.argtypes = [c_int, c_int, POINTER(c_int)]
    for name in EXPORTED_SYMBOLS:
        getattr(L, name)
    _lib = L
    return L


# ------------------------------------------------------------------ C-ABI mirrors (argument marshalling only)
def hb_status_string(status) -> str:
    return lib().hb_status_string(int(status)).decode()


def hb_last_error() -> str:
    return lib().hb_last_error().decode()


def hb_version() -> str:
    return lib().hb_version().decode()


def hb_device_peaks(cuda_device: int = 0):
    """measured pipe rates of the device: dict(ffma_tfma, dfma_tfma, tanh_tps, mma_f16_tflops, mma_tf32_tflops)"""
    out = (c_double * 5)()
    _check(lib().hb_device_peaks(int(cuda_device), out), "hb_device_peaks")
    return dict(zip(("ffma_tfma", "dfma_tfma", "tanh_tps", "mma_f16_tflops", "mma_tf32_tflops"), [float(v) for v in out]))


def hb_surrogate_kernel(prec, widths):
    """kernel a stage of this shape runs on ("fp32-ffma" | "tcgen05-resident" | "tcgen05-streamed"), None if unsupported"""
    w = (c_int * len(widths))(*[int(v) for v in widths])
    r = lib().hb_surrogate_kernel(PRECS[prec] if isinstance(prec, str) else int(prec), len(widths) - 1, w)
    return None if r is None else r.decode()


def _check(status, where):
    if status != 0:
        raise HbError(status, where)


def hb_lattice_create(ref_kinetic_energy_MeV: float, rest_energy_MeV: float):
    h = c_void_p()
    _check(lib().hb_lattice_create(ref_kinetic_energy_MeV, rest_energy_MeV, ctypes.byref(h)), "hb_lattice_create")
    return h


def hb_lattice_add_multipole(lat, order: int, kn: float, ks: float = 0.0):
    _check(lib().hb_lattice_add_multipole(lat, int(order), float(kn), float(ks)), "hb_lattice_add_multipole")


def hb_lattice_add_element(lat, kind, length_m: float = 0.0, param: float = 0.0):
    k = ELEM_KINDS[kind] if isinstance(kind, str) else int(kind)
    _check(lib().hb_lattice_add_element(lat, k, float(length_m), float(param)), "hb_lattice_add_element")


def hb_lattice_set_element(lat, index: int, length_m: float = 0.0, param: float = 0.0):
    _check(lib().hb_lattice_set_element(lat, int(index), float(length_m), float(param)), "hb_lattice_set_element")


def hb_lattice_add_surrogate(lat, widths, W, b, act, in_mean, in_std, out_mean, out_std, coord="s",
                             prelu_a=None, ref_bg_out=float("nan"), ref_z_out=float("nan"), prec="fp32"):
    nl = len(widths) - 1
    Wc = [np.ascontiguousarray(w, dtype=np.float32) for w in W]
    bc = [np.ascontiguousarray(x, dtype=np.float32) for x in b]
    if len(Wc) != nl or len(bc) != nl:
        raise ValueError("need %d weight matrices and biases" % nl)
    for l in range(nl):
        if Wc[l].shape != (widths[l + 1], widths[l]) or bc[l].shape != (widths[l + 1],):
            raise ValueError("layer %d: W must be [out,in]=%s, b [out]" % (l, (widths[l + 1], widths[l])))
    d = _SurrogateDesc()
    d.n_linear = nl
    wid = (c_int * (nl + 1))(*[int(w) for w in widths])
    d.widths = ctypes.cast(wid, POINTER(c_int))
    fp = POINTER(c_float)
    Wp = (fp * nl)(*[w.ctypes.data_as(fp) for w in Wc])
    bp = (fp * nl)(*[x.ctypes.data_as(fp) for x in bc])
    d.W = ctypes.cast(Wp, POINTER(fp))
    d.b = ctypes.cast(bp, POINTER(fp))
    d.act = ACTS[act] if isinstance(act, str) else int(act)
    a = None
    if prelu_a is not None:
        a = np.ascontiguousarray(prelu_a, dtype=np.float32)
        d.prelu_a = a.ctypes.data_as(fp)
    for name, src in (("in_mean", in_mean), ("in_std", in_std), ("out_mean", out_mean), ("out_std", out_std)):
        arr = getattr(d, name)
        for j in range(6):
            arr[j] = float(src[j])
    d.coord = COORDS[coord] if isinstance(coord, str) else int(coord)
    d.ref_bg_out = float(ref_bg_out)
    d.ref_z_out = float(ref_z_out)
    d.prec = PRECS[prec] if isinstance(prec, str) else int(prec)
    _check(lib().hb_lattice_add_surrogate(lat, ctypes.byref(d)), "hb_lattice_add_surrogate")


def hb_lattice_set_run_mode(lat, mode):
    m = RUN_MODES[mode] if isinstance(mode, str) else int(mode)
    _check(lib().hb_lattice_set_run_mode(lat, m), "hb_lattice_set_run_mode")


def hb_lattice_finalize(lat, cuda_device: int = 0):
    _check(lib().hb_lattice_finalize(lat, int(cuda_device)), "hb_lattice_finalize")


def hb_lattice_num_monitors(lat) -> int:
    n = c_int()
    _check(lib().hb_lattice_num_monitors(lat, ctypes.byref(n)), "hb_lattice_num_monitors")
    return n.value


def hb_lattice_num_launches(lat, with_moments: bool, n_particles: int) -> int:
    n = c_int()
    _check(lib().hb_lattice_num_launches(lat, int(bool(with_moments)), int(n_particles), ctypes.byref(n)),
           "hb_lattice_num_launches")
    return n.value


def hb_lattice_set_centroid(lat, centroid6):
    c = (c_double * 6)(*[float(v) for v in centroid6])
    _check(lib().hb_lattice_set_centroid(lat, c), "hb_lattice_set_centroid")


def hb_lattice_ref_bg_out(lat) -> float:
    v = c_double()
    _check(lib().hb_lattice_ref_bg_out(lat, ctypes.byref(v)), "hb_lattice_ref_bg_out")
    return v.value


def hb_push(lat, x, px, y, py, t, pt, n: int, cuda_stream: int = 0):
    """x..pt: device addresses (ints).  Enqueues on cuda_stream and returns."""
    _check(lib().hb_push(lat, x, px, y, py, t, pt, n, cuda_stream), "hb_push")


def hb_push_moments(lat, x, px, y, py, t, pt, n: int, d_moments: int, cuda_stream: int = 0):
    _check(lib().hb_push_moments(lat, x, px, y, py, t, pt, n, d_moments, cuda_stream), "hb_push_moments")


def hb_push_host(lat, x, px, y, py, t, pt, n: int, h_moments: int, chunks: int = 4):
    """x..pt, h_moments: HOST addresses (h_moments may be 0)"""
    _check(lib().hb_push_host(lat, x, px, y, py, t, pt, n, h_moments, int(chunks)), "hb_push_host")


def hb_push_candidates(lat, elem_index, length_m, param, x, px, y, py, t, pt, n: int, d_moments: int, cuda_stream: int = 0):
    """length_m, param: [K][n_set] (host); x..pt, d_moments: device addresses.  Enqueues on cuda_stream and returns."""
    idx = np.ascontiguousarray(elem_index, dtype=np.int32).reshape(-1)
    Lm = np.ascontiguousarray(length_m, dtype=np.float64).reshape(-1, idx.size)
    pm = np.ascontiguousarray(param, dtype=np.float64).reshape(-1, idx.size)
    if Lm.shape != pm.shape:
        raise ValueError("length_m and param must both be [K][n_set]")
    pd = POINTER(c_double)
    _check(lib().hb_push_candidates(lat, Lm.shape[0], idx.size, idx.ctypes.data_as(POINTER(c_int)), Lm.ctypes.data_as(pd),
                                    pm.ctypes.data_as(pd), x, px, y, py, t, pt, n, d_moments, cuda_stream),
           "hb_push_candidates")


def hb_moments_scratch_bytes() -> int:
    return int(lib().hb_moments_scratch_bytes())


def hb_moments(x, px, y, py, t, pt, n: int, pivot, d_out27: int, d_scratch: int, cuda_stream: int = 0):
    pv = None
    if pivot is not None:
        pv = (c_double * 6)(*[float(v) for v in pivot])
    _check(lib().hb_moments(x, px, y, py, t, pt, n, pv, d_out27, d_scratch, cuda_stream), "hb_moments")


def hb_moments_static_max_particles() -> int:
    return int(lib().hb_moments_static_max_particles())


def hb_moments_static(x, px, y, py, t, pt, n: int, pivot, d_out27: int, cuda_stream: int = 0):
    """hb_moments with the scratch in a static array of the library's device image: allocates nothing (include/hb.h)."""
    pv = None
    if pivot is not None:
        pv = (c_double * 6)(*[float(v) for v in pivot])
    _check(lib().hb_moments_static(x, px, y, py, t, pt, n, pv, d_out27, cuda_stream), "hb_moments_static")


def hb_moments_merge(rec_a, n_a: int, rec_b, n_b: int):
    """Record of the union of two disjoint particle sets (host arithmetic inside libhb.so).  rec_a / rec_b: 27 float64."""
    import numpy as np
    a = np.ascontiguousarray(rec_a, dtype=np.float64).reshape(27)
    b = np.ascontiguousarray(rec_b, dtype=np.float64).reshape(27)
    out = np.empty(27, dtype=np.float64)
    pd = POINTER(c_double)
    _check(lib().hb_moments_merge(a.ctypes.data_as(pd), int(n_a), b.ctypes.data_as(pd), int(n_b),
                                  out.ctypes.data_as(pd)), "hb_moments_merge")
    return out


def hb_lattice_enable_timing(lat, on: bool = True):
    _check(lib().hb_lattice_enable_timing(lat, int(bool(on))), "hb_lattice_enable_timing")


def hb_lattice_get_timing(lat):
    """milliseconds per segment of the most recent push (synchronises on its last event)"""
    cap = 4096
    buf = (c_float * cap)()
    n = c_int()
    _check(lib().hb_lattice_get_timing(lat, buf, cap, ctypes.byref(n)), "hb_lattice_get_timing")
    return [buf[i] for i in range(min(n.value, cap))]


def hb_lattice_destroy(lat):
    _check(lib().hb_lattice_destroy(lat), "hb_lattice_destroy")


# ------------------------------------------------------------------ torch plumbing (pointers + streams only)
def _rows(coords):
    """coords: torch float32 CUDA tensor [6, n] (rows contiguous) or a sequence of six 1-D tensors."""
    import torch
    rows = [coords[j] for j in range(6)]
    n = rows[0].numel()
    for r in rows:
        if not (isinstance(r, torch.Tensor) and r.is_cuda and r.dtype == torch.float32 and r.dim() == 1
                and r.is_contiguous() and r.numel() == n):
            raise ValueError("need six contiguous float32 CUDA vectors of equal length")
    return rows, n


def _stream(dev):
    import torch
    return torch.cuda.current_stream(dev).cuda_stream


def to_device(x, device="cuda"):
    """numpy/torch [6, n] float32 -> list of six 16-byte-aligned CUDA row views (row pitch padded to 4 floats)."""
    import torch
    t = torch.as_tensor(x, dtype=torch.float32)
    n = t.shape[1]
    pitch = (n + 3) // 4 * 4
    buf = torch.zeros((6, max(pitch, 4)), dtype=torch.float32, device=device)
    buf[:, :n] = t.to(device)
    return [buf[j, :n] for j in range(6)]


def to_host(rows):
    import torch
    return torch.stack([r for r in rows]).cpu().numpy()


class Lattice:
    """Owning wrapper of an hb_lattice.  `Lattice.from_description(desc)` consumes the plain-data lattice
    description of workloads/ (also consumed, independently, by the oracle)."""

    def __init__(self, kinetic_MeV: float, rest_MeV: float):
        self._h = hb_lattice_create(kinetic_MeV, rest_MeV)
        self.device = None

    @classmethod
    def from_description(cls, desc, run_mode="composed", device=0, prec=None, finalize=True):
        lat = cls(desc["kinetic_MeV"], desc["rest_MeV"])
        for el in desc["elements"]:
            k = el["kind"]
            if k in ("drift", "drift_exact"):
                lat.add_element(k, el["L"])
            elif k in ("quad", "plens", "quad_chromatic"):
                lat.add_element(k, el["L"], el["k"])
            elif k == "multipole":
                hb_lattice_add_multipole(lat._h, el["order"], el["kn"], el["ks"])
            elif k == "sbend":
                lat.add_element("sbend", el["L"], el["theta"])
            elif k == "monitor":
                lat.add_element("monitor")
            elif k == "surrogate":
                lat.add_surrogate(el["widths"], el["W"], el["b"], el["act"], el["in_mean"], el["in_std"],
                                  el["out_mean"], el["out_std"], coord=el["coord"], prelu_a=el.get("prelu_a"),
                                  ref_bg_out=el["ref_bg_out"], ref_z_out=el["ref_z_out"],
                                  prec=prec if prec is not None else el["prec"])
            else:
                raise ValueError(k)
        lat.set_run_mode(run_mode)
        if finalize:
            lat.finalize(device)
        return lat

    def add_element(self, kind, length_m=0.0, param=0.0):
        hb_lattice_add_element(self._h, kind, length_m, param)

    def set_element(self, index, length_m=0.0, param=0.0):
        """re-set length / parameter of element `index` (position in the description's element list)"""
        hb_lattice_set_element(self._h, index, length_m, param)

    def add_surrogate(self, *a, **k):
        hb_lattice_add_surrogate(self._h, *a, **k)

    def set_run_mode(self, mode):
        hb_lattice_set_run_mode(self._h, mode)

    def finalize(self, device=0):
        hb_lattice_finalize(self._h, device)
        self.device = device

    @property
    def num_monitors(self):
        return hb_lattice_num_monitors(self._h)

    def num_launches(self, with_moments, n_particles):
        return hb_lattice_num_launches(self._h, with_moments, n_particles)

    def set_centroid(self, centroid6):
        """nominal centroid of the incoming bunch (pivot of the moment sums; default zeros)"""
        hb_lattice_set_centroid(self._h, centroid6)

    @property
    def ref_bg_out(self):
        return hb_lattice_ref_bg_out(self._h)

    def push(self, coords):
        rows, n = _rows(coords)
        hb_push(self._h, *[r.data_ptr() for r in rows], n, _stream(rows[0].device))

    def push_moments(self, coords, out=None):
        import torch
        rows, n = _rows(coords)
        m = self.num_monitors
        if out is None:
            out = torch.empty((m, 27), dtype=torch.float64, device=rows[0].device)
        hb_push_moments(self._h, *[r.data_ptr() for r in rows], n, out.data_ptr(), _stream(rows[0].device))
        return out

    def push_candidates(self, coords, elem_index, length_m, param, out=None):
        """records [K, 27] of the bunch `coords` (as it enters the run that holds `elem_index`) behind that run, for K
        settings (length_m, param: [K][n_set]) of those elements; the bunch and the lattice are not changed"""
        import torch
        rows, n = _rows(coords)
        k = int(np.asarray(length_m).reshape(-1, len(elem_index)).shape[0])
        if out is None:
            out = torch.empty((k, 27), dtype=torch.float64, device=rows[0].device)
        hb_push_candidates(self._h, elem_index, length_m, param, *[r.data_ptr() for r in rows], n, out.data_ptr(),
                           _stream(rows[0].device))
        return out

    def push_host(self, host_coords, chunks=4, moments=True):
        """host_coords: CPU float32 tensor or numpy array [6, n] (C-contiguous rows; pinned memory overlaps the copies);
        pushed in place through hb_push_host; returns the [num_monitors, 27] records (numpy) or None"""
        import numpy as np
        rows = [host_coords[j] for j in range(6)]
        n = int(rows[0].shape[0])
        ptrs = [int(r.data_ptr()) if hasattr(r, "data_ptr") else int(r.ctypes.data) for r in rows]
        rec = np.empty((self.num_monitors, 27), dtype=np.float64) if (moments and self.num_monitors) else None
        hb_push_host(self._h, *ptrs, n, 0 if rec is None else rec.ctypes.data, chunks)
        return rec

    def enable_timing(self, on=True):
        hb_lattice_enable_timing(self._h, on)

    def segment_times_ms(self):
        return hb_lattice_get_timing(self._h)

    def close(self):
        if self._h is not None:
            hb_lattice_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


_scratch = {}


def moments(coords, pivot=None, out=None):
    """Standalone bunch moments (27 doubles, R10) of a [6,n] float32 CUDA tensor."""
    import torch
    rows, n = _rows(coords)
    dev = rows[0].device
    if out is None:
        out = torch.empty(27, dtype=torch.float64, device=dev)
    key = (dev.index, _stream(dev))
    if key not in _scratch:
        _scratch[key] = torch.empty(hb_moments_scratch_bytes(), dtype=torch.uint8, device=dev)
    hb_moments(*[r.data_ptr() for r in rows], n, pivot, out.data_ptr(), _scratch[key].data_ptr(), _stream(dev))
    return out


def moments_static(coords, out, pivot=None):
    """As moments(), through hb_moments_static: the caller owns `out` (27 float64 on the bunch's device), the scratch is
    the library's static device array, nothing is allocated.  Calls that overlap on the GPU race on that array."""
    rows, n = _rows(coords)
    dev = rows[0].device
    hb_moments_static(*[r.data_ptr() for r in rows], n, pivot, out.data_ptr(), _stream(dev))
    return out


def allgather_merge_records(records, n_local: int, group=None):
    """Monitor records of a bunch sharded over the ranks of a torch.distributed group (each rank pushes its own
    particles; no other exchange on the path).  records: [m, 27] float64 (tensor or array) of this rank's shard,
    n_local its particle count.  All-gathers the m records and counts (224 B per monitor and rank) and merges them
    in rank order with hb_moments_merge, so every rank returns the same [m, 27] numpy array: the records of the
    whole bunch."""
    import numpy as np
    import torch
    import torch.distributed as dist
    rec = torch.as_tensor(records).detach().to("cpu", torch.float64).reshape(-1, 27).contiguous()
    m = rec.shape[0]
    if not (dist.is_available() and dist.is_initialized()):
        return rec.numpy().copy()
    world = dist.get_world_size(group)
    backend = dist.get_backend(group)
    dev = torch.device("cuda", torch.cuda.current_device()) if backend == "nccl" else torch.device("cpu")
    # counts travel as two 32-bit halves inside the float64 payload (exact for any size_t below 2^64)
    mine = torch.empty(m * 27 + 2, dtype=torch.float64)
    mine[:m * 27] = rec.reshape(-1)
    mine[m * 27] = float(int(n_local) >> 32)
    mine[m * 27 + 1] = float(int(n_local) & 0xffffffff)
    mine = mine.to(dev)
    parts = [torch.empty_like(mine) for _ in range(world)]
    dist.all_gather(parts, mine, group=group)
    parts = [q.cpu().numpy() for q in parts]
    out = np.empty((m, 27), dtype=np.float64)
    for k in range(m):
        acc, n_acc = None, 0
        for q in parts:
            n_q = (int(q[m * 27]) << 32) | int(q[m * 27 + 1])
            r_q = q[k * 27:(k + 1) * 27]
            if acc is None:
                acc, n_acc = r_q.copy(), n_q
            else:
                acc = hb_moments_merge(acc, n_acc, r_q, n_q)
                n_acc += n_q
        out[k] = acc
    return out
