"""GPU-vs-oracle parity through the C ABI (run with -m gpu on a B200).

Tolerances (BASELINE.json north_star): max |gpu - oracle| <= 1e-6 x std(oracle coordinate) for fp32
element maps, <= 1e-5 for the fp32 surrogate path, <= 2e-2 for the 16-bit tensor-core path; moments
within 1e-4 relative.  "std" = centred std of the oracle's output coordinate (G14).
"""
import math

import numpy as np
import pytest

import oracle
import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def hb():
    import torch
    assert torch.cuda.is_available()
    import paper_2402_17248_b200 as hb
    hb.lib()
    return hb


def gpu_push(hb, desc, x, run_mode="composed", moments=True, prec=None):
    import torch
    lat = hb.Lattice.from_description(desc, run_mode=run_mode, device=0, prec=prec)
    c = hb.to_device(x)
    rec = None
    if moments:
        rec = lat.push_moments(c)
    else:
        lat.push(c)
    torch.cuda.synchronize()
    out = hb.to_host(c).astype(np.float64)
    rec = None if rec is None else rec.cpu().numpy()
    lat.close()
    return out, rec


def rel_err(got, ref):
    return np.max(np.abs(got - ref), axis=1) / ref.std(axis=1)


def sym(rec):
    C = np.zeros((6, 6))
    C[np.triu_indices(6)] = rec[6:]
    return C + C.T - np.diag(np.diag(C))


def moments_close(rec, ref, tol):
    """means relative to sigma, second moments relative to sqrt(C_jj C_kk)"""
    C, R = sym(rec), sym(ref)
    sd = np.sqrt(np.diag(R))
    assert np.max(np.abs(rec[:6] - ref[:6]) / sd) <= tol
    assert np.max(np.abs(C - R) / np.outer(sd, sd)) <= tol


# --------------------------------------------------------------------------------- a2: conventional runs
@pytest.mark.parametrize("mode,tol", [("composed", 1e-6), ("sequential", 1e-6)])
@pytest.mark.parametrize("n", [1, 3, 4, 5, 1023, 4096, 100003])
def test_run_parity_small(hb, mode, tol, n):
    desc = wl.lattice(wl.fodo_cell(1.0) + wl.c4_transport() + [wl.monitor()])
    x = wl.gaussian_bunch(max(n, 8), 11)[:, :n].copy()
    ref, ref_rec = oracle.push(desc, x)
    got, rec = gpu_push(hb, desc, x, run_mode=mode)
    if n >= 1000:
        assert rel_err(got, ref).max() <= tol
        moments_close(rec[0], ref_rec[0], 1e-4)
    else:
        scale = wl.NOMINAL_SIGMA[:, None] * 5
        assert np.max(np.abs(got - ref) / scale) <= tol


@pytest.mark.parametrize("mode", ["composed", "sequential"])
def test_config2_parity_and_emittance(hb, mode):
    desc, x = wl.config2()
    ref, ref_rec = oracle.push(desc, x)
    got, rec = gpu_push(hb, desc, x, run_mode=mode)
    e = rel_err(got, ref)
    print("C2", mode, "max err/std per coordinate:", e)
    assert e.max() <= 1e-6
    moments_close(rec[0], ref_rec[0], 1e-4)
    # the GPU's fused fp64 moments equal the fp64 moments of the GPU's own fp32 output (pure reduction check)
    own = oracle.moments(np.ascontiguousarray(got))
    moments_close(rec[0], own, 1e-10)
    # rms emittance from the GPU record vs oracle
    for j in (0, 2):
        C, R = sym(rec[0]), sym(ref_rec[0])
        eg = math.sqrt(C[j, j] * C[j + 1, j + 1] - C[j, j + 1] ** 2)
        eo = math.sqrt(R[j, j] * R[j + 1, j + 1] - R[j, j + 1] ** 2)
        assert abs(eg / eo - 1) <= 1e-4


def test_sequential_fp32_reported_not_bounded(hb):
    """HB_RUN_SEQUENTIAL_FP32 is the literal 'fp32 registers' reading; its error grows with run length
    (DESIGN.md): report it, require only that it stays within 2e-4 over 500 elements."""
    desc, x = wl.config2(n=200_000)
    ref, _ = oracle.push(desc, x)
    got, _ = gpu_push(hb, desc, x, run_mode="sequential_fp32", moments=False)
    e = rel_err(got, ref)
    print("C2 sequential_fp32 max err/std:", e)
    assert e.max() <= 2e-4


def test_drift_roundtrip_identity_on_gpu(hb):
    desc = wl.lattice([wl.drift(0.7), wl.drift(-0.7)])
    x = wl.gaussian_bunch(4096, 5)
    got, _ = gpu_push(hb, desc, x, moments=False)
    assert np.array_equal(got.astype(np.float32), x)          # composed run = identity matrix exactly
    got, _ = gpu_push(hb, desc, x, run_mode="sequential", moments=False)
    assert np.max(np.abs(got - x) / wl.NOMINAL_SIGMA[:, None]) < 1e-6


def test_long_run_500_elements_and_single_element(hb):
    desc = wl.lattice([wl.quad(0.1, 1.2)])
    x = wl.gaussian_bunch(5000, 6)
    ref, _ = oracle.push(desc, x)
    for mode in ("composed", "sequential"):
        got, _ = gpu_push(hb, desc, x, run_mode=mode, moments=False)
        assert rel_err(got, ref).max() <= 1e-6


# --------------------------------------------------------------------------------- a3: moments
@pytest.mark.parametrize("n", [1, 2, 7, 4096, 1_000_003])
def test_standalone_moments(hb, n):
    import torch
    x = wl.gaussian_bunch(max(n, 8), 21)[:, :n].copy() + (np.arange(6, dtype=np.float32)[:, None] * 1e-3)
    ref = oracle.moments(np.ascontiguousarray(x.astype(np.float64)))
    c = hb.to_device(x)
    for pivot in (None, list(np.arange(6) * 1e-3)):
        rec = hb.moments(c, pivot=pivot).cpu().numpy()
        assert np.allclose(rec[:6], ref[:6], rtol=1e-12, atol=1e-18)
        if n > 1:
            C, R = sym(rec), sym(ref)
            sd = np.sqrt(np.diag(R))
            assert np.max(np.abs(C - R) / np.outer(sd, sd)) < 1e-9
    assert np.array_equal(hb.to_host(c), x)                   # read-only


def test_monitor_without_producer_and_double_monitor(hb):
    desc = wl.lattice([wl.monitor(), wl.drift(1.0), wl.monitor(), wl.monitor()])
    x = wl.gaussian_bunch(10_001, 8)
    ref, ref_rec = oracle.push(desc, x)
    got, rec = gpu_push(hb, desc, x)
    assert rec.shape == (3, 27)
    for k in range(3):
        moments_close(rec[k], ref_rec[k], 1e-6)
    assert np.allclose(rec[1], rec[2], rtol=1e-12, atol=1e-30)


# --------------------------------------------------------------------------------- a4-a6: fp32 surrogate
def test_config1_fp32_per_segment(hb):
    desc, x = wl.config1(prec="fp32")
    states = []
    ref, ref_rec = oracle.push(desc, x, on_element=lambda i, el, c: states.append(c.copy()) if el["kind"] == "monitor" else None)
    got, rec = gpu_push(hb, desc, x)
    e = rel_err(got, ref)
    print("C1 fp32 end-to-end err/std:", e)
    assert e.max() <= 1e-5
    for k in range(3):
        moments_close(rec[k], ref_rec[k], 1e-4)
    # segment 1 alone (conventional): 1e-6
    cell = wl.lattice(desc["elements"][:5])
    g1, _ = gpu_push(hb, cell, x, moments=False)
    assert rel_err(g1, states[0]).max() <= 1e-6


@pytest.mark.parametrize("act", ["identity", "relu", "prelu", "tanh"])
@pytest.mark.parametrize("widths", [[6, 6], [6, 7, 6], [6, 64, 64, 6], [6, 100, 37, 6], [6, 256, 256, 256, 6],
                                    [6, 200, 256, 6], [6, 320, 192, 6], [6, 128, 128, 6]])
def test_fp32_surrogate_shapes(hb, act, widths):
    n = 3001
    W, b = wl.make_mlp(widths, "he" if act in ("relu", "prelu") else "xavier", 77, len(widths))
    rng = np.random.default_rng(5)
    a = rng.uniform(0.05, 0.3, len(widths) - 2).astype(np.float32) if act == "prelu" else None
    sur = wl.surrogate(widths, W, b, act, rng.normal(size=6) * 1e-4, wl.NOMINAL_SIGMA, rng.normal(size=6),
                       rng.uniform(0.5, 2.0, 6), prelu_a=a)
    desc = wl.lattice([sur, wl.monitor()])
    x = wl.gaussian_bunch(n, 31)
    ref, ref_rec = oracle.push(desc, x)
    got, rec = gpu_push(hb, desc, x)
    e = rel_err(got, ref)
    assert e.max() <= 1e-5, e
    moments_close(rec[0], ref_rec[0], 1e-4)


@pytest.mark.parametrize("widths", [[6, 256, 256, 6], [6, 128, 128, 128, 6]])
def test_fp32_register_tile_shapes_agree(hb, widths, monkeypatch):
    """The 8x8-register-tile shapes (256- / 128-wide output blocks) and the 4x4 shape (forced with HB_FP32_TP, read by
    the library at launch) are two schedules of the same sums: both within the fp32 bound of the oracle, and the
    hidden-layer summation order is the same, so they differ only through the output layer's K split."""
    n = 64 * 37 + 5
    W, b = wl.make_mlp(widths, "xavier", 91, len(widths))
    rng = np.random.default_rng(8)
    sur = wl.surrogate(widths, W, b, "tanh", rng.normal(size=6) * 1e-4, wl.NOMINAL_SIGMA, rng.normal(size=6),
                       rng.uniform(0.5, 2.0, 6))
    desc = wl.lattice([sur, wl.monitor()])
    x = wl.gaussian_bunch(n, 32)
    ref, ref_rec = oracle.push(desc, x)
    got8, rec8 = gpu_push(hb, desc, x)
    monkeypatch.setenv("HB_FP32_TP", "32")
    got4, rec4 = gpu_push(hb, desc, x)
    monkeypatch.delenv("HB_FP32_TP")
    assert rel_err(got8, ref).max() <= 1e-5 and rel_err(got4, ref).max() <= 1e-5
    assert rel_err(got8, got4.astype(np.float64)).max() <= 2e-6
    moments_close(rec8[0], ref_rec[0], 1e-4)
    moments_close(rec4[0], ref_rec[0], 1e-4)


def test_fp32_identity_initialised_net(hb):
    H = 64
    A0 = np.zeros((H, 6), np.float32); A0[:6] = np.eye(6)
    A1 = np.zeros((H, H), np.float32); A1[:6, :6] = np.eye(6)
    A2 = np.zeros((6, H), np.float32); A2[:, :6] = np.eye(6)
    zb = [np.zeros(H, np.float32), np.zeros(H, np.float32), np.zeros(6, np.float32)]
    z, o = np.zeros(6), np.ones(6)
    sur = wl.surrogate([6, H, H, 6], [A0, A1, A2], zb, "prelu", z, o, z, o, prelu_a=[1.0, 1.0])
    x = wl.gaussian_bunch(1000, 3, sigma=np.ones(6))
    got, _ = gpu_push(hb, wl.lattice([sur]), x, moments=False)
    assert np.array_equal(got.astype(np.float32), x)


def test_fp32_coord_t_stage(hb):
    desc, x = wl.config4(prec="fp32", n=20_000, stages=2)
    ref, ref_rec = oracle.push(desc, x)
    got, rec = gpu_push(hb, desc, x)
    assert np.all(np.isfinite(got))
    e = rel_err(got, ref)
    print("C4 fp32 (2 stages, free running) err/std:", e)
    assert e.max() <= 1e-4       # two stages compound; the per-stage bound is checked below
    # per-stage: stage 1 only
    d1 = wl.lattice(desc["elements"][:1])
    r1, _ = oracle.push(d1, x)
    g1, _ = gpu_push(hb, d1, x, moments=False)
    e1 = rel_err(g1, r1)
    print("C4 fp32 stage 1 err/std:", e1)
    assert e1.max() <= 1e-5
    for k in range(4):
        moments_close(rec[k], ref_rec[k], 1e-4)


def test_cross_pin_linear_surrogate_equals_run_kernel(hb):
    """ties a5 to a2: identity-activation 1-layer surrogate with A = D^-1 M D reproduces the run kernel."""
    els = wl.fodo_cell(1.2)
    c = np.zeros((6, 6)); c[:] = np.eye(6)
    M, _ = oracle.push(wl.lattice(els), c)
    sd = wl.NOMINAL_SIGMA
    A = (np.diag(1 / sd) @ M @ np.diag(sd)).astype(np.float32)
    sur = wl.surrogate([6, 6], [A], [np.zeros(6, np.float32)], "identity", np.zeros(6), sd, np.zeros(6), sd)
    x = wl.gaussian_bunch(4096, 9)
    g_run, _ = gpu_push(hb, wl.lattice(els), x, moments=False)
    g_sur, _ = gpu_push(hb, wl.lattice([sur]), x, moments=False)
    assert np.max(np.abs(g_run - g_sur) / sd[:, None]) < 2e-6


# --------------------------------------------------------------------------------- boundary behaviour
def test_abi_errors(hb):
    import torch
    lat = hb.Lattice(1000.0, wl.ELECTRON_MEV)
    lat.add_element("drift", 1.0)
    c = torch.zeros((6, 16), dtype=torch.float32, device="cuda")
    with pytest.raises(hb.HbError) as ei:
        lat.push(c)                                            # not finalized
    assert ei.value.status == 2
    lat.finalize(0)
    with pytest.raises(hb.HbError) as ei:
        lat.add_element("drift", 1.0)                          # finalized
    assert ei.value.status == 2
    lat.push(c)
    big = torch.zeros(6 * 16 + 1, dtype=torch.float32, device="cuda")
    mis = [big[1 + 16 * j: 1 + 16 * (j + 1)] for j in range(6)]   # 4-byte offset: misaligned
    with pytest.raises(hb.HbError) as ei:
        lat.push(mis)
    assert ei.value.status == 1
    alias = [c[0], c[0], c[2], c[3], c[4], c[5]]
    with pytest.raises(hb.HbError) as ei:
        lat.push(alias)
    assert ei.value.status == 1
    e = torch.zeros((6, 0), dtype=torch.float32, device="cuda")
    lat.push(e)                                                # n = 0 is a no-op
    lat.close()
    with pytest.raises(hb.HbError):
        hb.hb_lattice_create(-1.0, 0.511)
    h = hb.hb_lattice_create(1000.0, 0.511)
    with pytest.raises(hb.HbError):
        hb.hb_lattice_add_element(h, "quad", -0.1, 1.0)
    with pytest.raises(hb.HbError):
        hb.hb_lattice_add_surrogate(h, [6, 8, 5], [np.zeros((8, 6), np.float32), np.zeros((5, 8), np.float32)],
                                    [np.zeros(8, np.float32), np.zeros(5, np.float32)], "relu",
                                    np.zeros(6), np.ones(6), np.zeros(6), np.ones(6))
    hb.hb_lattice_destroy(h)


def test_stream_ordering_and_inplace(hb):
    import torch
    desc = wl.lattice(wl.fodo_cell(1.2))
    x = wl.gaussian_bunch(50_000, 13)
    ref, _ = oracle.push(wl.lattice(wl.fodo_cell(1.2) * 2), x)
    lat = hb.Lattice.from_description(desc, device=0)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        c = torch.from_numpy(x).cuda()
        lat.push(c)
        lat.push(c)                                            # back-to-back on a non-default stream
    s.synchronize()
    got = c.cpu().numpy().astype(np.float64)
    assert rel_err(got, ref).max() <= 2e-6
    lat.close()


def test_push_is_capturable_in_a_cuda_graph(hb):
    """row a7: hb_push_moments only enqueues work on the caller's stream (no host sync, no allocation), so a whole
    hybrid lattice (runs, tensor-core surrogate, monitors) can be captured once in a CUDA graph and replayed"""
    import torch
    desc, x = wl.config1(prec="f16", n=3000)
    ref, ref_rec = oracle.push(desc, x)
    lat = hb.Lattice.from_description(desc, device=0)
    pristine = torch.from_numpy(x).cuda()
    work = torch.empty_like(pristine)
    rec = torch.zeros((lat.num_monitors, 27), dtype=torch.float64, device="cuda")
    work.copy_(pristine)
    lat.push_moments(work, out=rec)              # warm-up outside the capture (cudaFuncSetAttribute etc.)
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        work.copy_(pristine)
        lat.push_moments(work, out=rec)
    for _ in range(3):
        rec.zero_()
        g.replay()
    torch.cuda.synchronize()
    got = work.cpu().numpy().astype(np.float64)
    assert rel_err(got, ref).max() <= 2e-2
    own = oracle.moments(np.ascontiguousarray(got))
    assert np.allclose(rec[-1].cpu().numpy()[:6], own[:6], rtol=1e-9, atol=1e-16)
    lat.close()


# ------------------------------------------------------------------ NEXT-2: plasma lens + moments -> host feedback
@pytest.mark.parametrize("mode,tol", [("composed", 1e-6), ("sequential", 1e-6)])
def test_plasma_lens_runs(hb, mode, tol):
    """thick axisymmetric lens (R3b) inside fused runs: focusing, defocusing, zero strength, between other elements"""
    els = [wl.drift(0.3), wl.plens(0.05, 40.0), wl.drift(0.2), wl.quad(0.1, 1.2), wl.plens(0.02, -15.0),
           wl.sbend(0.5, 0.02), wl.plens(0.1, 0.0), wl.plens(0.03, 400.0), wl.drift(0.1), wl.monitor()]
    desc = wl.lattice(els)
    x = wl.gaussian_bunch(100_003, 21)
    ref, ref_rec = oracle.push(desc, x)
    got, rec = gpu_push(hb, desc, x, run_mode=mode, moments=True)
    assert rel_err(got, ref).max() <= tol
    diag = [6, 12, 17, 21, 24, 26]
    assert np.allclose(rec[0][diag], ref_rec[0][diag], rtol=1e-4)


def lens_strength_from_record(rec):
    """a caller-side rule (the paper's own expression is in its ref. [31], not in the paper): matched focusing for
    the measured beam, k = (eps/sigma^2)^2 averaged over the two planes, times a fixed factor"""
    sxx, sxpx, spxpx = rec[6], rec[7], rec[12]
    syy, sypy, spypy = rec[17], rec[18], rec[21]
    ex2, ey2 = sxx * spxpx - sxpx ** 2, syy * spypy - sypy ** 2
    return 50.0 * 0.5 * (ex2 / sxx ** 2 + ey2 / syy ** 2)


def test_moments_to_host_feedback_sets_the_lens(hb):
    """the paper's in-situ lens setting: push a stage, read the moment record on the host, set the strength
    of the following plasma lens from it, push the transport -- on the GPU and in the oracle, same rule"""
    import torch
    desc1, x = wl.config1(prec="fp32", n=50_000)
    stage = wl.lattice(desc1["elements"][:8])                      # FODO cell | monitor | surrogate | monitor
    ref1, ref_rec1 = oracle.push(stage, x)
    k_ref = lens_strength_from_record(ref_rec1[-1])
    gap_ref = wl.lattice([wl.drift(0.1), wl.plens(0.02, k_ref), wl.drift(0.1), wl.monitor()])
    ref2, ref_rec2 = oracle.push(gap_ref, ref1.astype(np.float32))

    lat1 = hb.Lattice.from_description(stage, device=0)
    c = hb.to_device(x)
    rec1 = lat1.push_moments(c)
    torch.cuda.synchronize()                                       # the per-stage device -> host sync the paper has
    k_gpu = lens_strength_from_record(rec1[-1].cpu().numpy())
    assert abs(k_gpu - k_ref) <= 1e-4 * abs(k_ref) and k_gpu > 0
    lat2 = hb.Lattice.from_description(wl.lattice([wl.drift(0.1), wl.plens(0.02, k_gpu), wl.drift(0.1), wl.monitor()]), device=0)
    rec2 = lat2.push_moments(c)
    torch.cuda.synchronize()
    got = hb.to_host(c).astype(np.float64)
    assert rel_err(got, ref2).max() <= 2e-5
    diag = [6, 12, 17, 21, 24, 26]
    assert np.allclose(rec2[-1].cpu().numpy()[diag], ref_rec2[-1][diag], rtol=1e-4)
    lat1.close(); lat2.close()


# ------------------------------------------------------------------ NEXT-3: non-linear map in sequential mode
@pytest.mark.parametrize("mode", ["composed", "sequential", "sequential_fp32"])
def test_exact_drift_runs_in_fp64_registers_whatever_the_mode(hb, mode):
    """a run holding a non-linear element (exact drift R2x) has no composed matrix: it always goes element by element
    through the fp64 sequential kernel; large divergences and momentum offsets make the non-linearity matter"""
    sig = np.array([1e-3, 2e-2, 1e-3, 2e-2, 1e-3, 3e-2])
    x = wl.gaussian_bunch(70_001, 23, sigma=sig)
    els = [wl.drift_exact(0.8), wl.quad(0.1, 1.2), wl.drift_exact(1.5), wl.plens(0.02, 30.0), wl.drift_exact(-0.3),
           wl.sbend(0.5, 0.02), wl.drift(0.2), wl.monitor()]
    desc = wl.lattice(els)
    ref, ref_rec = oracle.push(desc, x)
    lin, _ = oracle.push(wl.lattice([wl.drift(e["L"]) if e["kind"] == "drift_exact" else e for e in els]), x)
    assert rel_err(lin, ref).max() > 1e-3                      # the paraxial drift is visibly different here
    got, rec = gpu_push(hb, desc, x, run_mode=mode, moments=True)
    assert rel_err(got, ref).max() <= 1e-6
    diag = [6, 12, 17, 21, 24, 26]
    assert np.allclose(rec[0][diag], ref_rec[0][diag], rtol=1e-4)


def test_chromatic_quads_and_multipole_kicks(hb):
    """the rest of NEXT-3: a chromatic FODO cell (exact drifts + momentum-dependent quadrupoles) with sextupole /
    octupole / skew kicks, wide momentum spread, against the oracle; and the first-order limit on the device:
    on-momentum, small amplitudes -> the linear cell of the composed kernel"""
    sig = np.array([1e-3, 1e-3, 1e-3, 1e-3, 1e-3, 3e-2])
    x = wl.gaussian_bunch(60_007, 29, sigma=sig)
    els = [wl.drift_exact(0.25), wl.quad_chromatic(0.1, 1.2), wl.multipole(3, 20.0, -5.0), wl.drift_exact(0.5),
           wl.quad_chromatic(0.1, -1.2), wl.multipole(4, 3e3, 1e3), wl.multipole(1, 1e-5, -2e-5), wl.drift_exact(0.25),
           wl.quad_chromatic(0.2, 0.0), wl.multipole(2, 0.1, 0.05), wl.monitor()]
    desc = wl.lattice(els)
    ref, ref_rec = oracle.push(desc, x)
    got, rec = gpu_push(hb, desc, x, run_mode="composed", moments=True)
    assert np.all(np.isfinite(got))
    assert rel_err(got, ref).max() <= 1e-6
    diag = [6, 12, 17, 21, 24, 26]
    assert np.allclose(rec[0][diag], ref_rec[0][diag], rtol=1e-4)
    # chromaticity is visible: the linear cell differs at the per-cent level for this momentum spread
    lin_els = wl.fodo_cell(1.2) + [wl.drift(0.2), wl.monitor()]
    lin, _ = oracle.push(wl.lattice(lin_els), x)
    assert rel_err(lin, ref).max() > 1e-2
    # first-order limit on the device
    small = wl.gaussian_bunch(10_000, 31, sigma=np.array([1e-6, 1e-7, 1e-6, 1e-7, 1e-6, 1e-9]))
    chrom = [wl.drift_exact(0.25), wl.quad_chromatic(0.1, 1.2), wl.drift_exact(0.5), wl.quad_chromatic(0.1, -1.2),
             wl.drift_exact(0.25)]
    a, _ = gpu_push(hb, wl.lattice(chrom), small, moments=False)
    b, _ = gpu_push(hb, wl.lattice(wl.fodo_cell(1.2)), small, moments=False)
    assert np.max(np.abs(a - b) / b.std(axis=1)[:, None]) <= 2e-6


def test_multipole_validation(hb):
    h = hb.hb_lattice_create(1000.0, wl.ELECTRON_MEV)
    hb.hb_lattice_add_multipole(h, 3, 1.0, 0.0)
    for bad in ((0, 1.0, 0.0), (9, 1.0, 0.0), (2, float("nan"), 0.0)):
        with pytest.raises(hb.HbError):
            hb.hb_lattice_add_multipole(h, *bad)
    with pytest.raises(hb.HbError):
        hb.hb_lattice_add_element(h, 8, 0.0, 1.0)          # a multipole needs its own call
    hb.hb_lattice_destroy(h)


# ------------------------------------------------------------------ hb_push_host: host-resident bunch, chunked pipeline
@pytest.mark.parametrize("chunks", [1, 2, 3, 8])
@pytest.mark.parametrize("n", [1, 255, 70_001])
def test_push_host_equals_device_push(hb, chunks, n):
    """the host entry point runs the same kernels piece by piece: coordinates bit-identical to hb_push_moments on the
    whole bunch, records equal up to the summation order of the partials"""
    import torch
    desc, x = wl.config1(prec="f16", n=max(n, 8))
    x = np.ascontiguousarray(x[:, :n])
    lat = hb.Lattice.from_description(desc, device=0)
    c = hb.to_device(x)
    rec_dev = lat.push_moments(c)
    torch.cuda.synchronize()
    dev = hb.to_host(c)
    host = torch.from_numpy(x.copy()).pin_memory()
    rec_host = lat.push_host(host, chunks=chunks)
    assert np.array_equal(host.numpy(), dev)
    r = rec_dev.cpu().numpy()
    assert np.allclose(rec_host[:, :6], r[:, :6], rtol=1e-12, atol=1e-18)
    if n > 1:
        diag = [6, 12, 17, 21, 24, 26]
        assert np.allclose(rec_host[:, diag], r[:, diag], rtol=1e-10)
    # pageable numpy memory works too (copies are then synchronous), and so does a second call on the same lattice
    again = x.copy()
    rec2 = lat.push_host(again, chunks=chunks)
    assert np.array_equal(again, dev) and np.allclose(rec2[:, :6], r[:, :6], rtol=1e-12, atol=1e-18)
    lat.close()


def test_push_host_vs_oracle_and_errors(hb):
    import torch
    desc, x = wl.config4(prec="f16", n=120_000)
    ref, ref_rec = oracle.push(desc, x)
    lat = hb.Lattice.from_description(desc, device=0)
    host = torch.from_numpy(x.copy()).pin_memory()
    rec = lat.push_host(host, chunks=4)
    got = host.numpy().astype(np.float64)
    assert rel_err(got, ref).max() <= 5e-2
    own = oracle.moments(np.ascontiguousarray(got))
    assert np.allclose(rec[-1][:6], own[:6], rtol=1e-9, atol=1e-16)
    diag = [6, 12, 17, 21, 24, 26]
    assert np.allclose(rec[-1][diag], own[diag], rtol=1e-9)
    assert lat.push_host(host, chunks=2, moments=False) is None
    with pytest.raises(hb.HbError):
        lat.push_host(host, chunks=0)
    with pytest.raises(hb.HbError):
        lat.push_host(host, chunks=9)
    empty = np.zeros((6, 0), np.float32)
    r0 = lat.push_host(empty, chunks=1)
    assert np.all(np.isnan(r0))
    lat.close()


def test_lens_optimisation_loop_on_the_gpu(hb):
    """NEXT-4 in miniature (the paper's headline use is an optimiser around the beamline): Nelder-Mead
    over the strengths of two plasma lenses, every objective evaluation = one lattice build + one hb_push_moments of
    a 1e5-particle bunch on the GPU; the optimum is then checked with the fp64 oracle"""
    import torch
    from scipy.optimize import minimize
    x = wl.gaussian_bunch(100_000, 37, sigma=np.array([1e-3, 1e-3, 1e-3, 1e-3, 1e-3, 1e-3]))
    c0 = torch.from_numpy(x).cuda()
    work = torch.empty_like(c0)

    def line(k):
        return wl.lattice([wl.drift(0.5), wl.plens(0.05, k[0]), wl.drift(1.0), wl.plens(0.05, k[1]), wl.drift(0.7), wl.monitor()])

    evals = []

    def objective(k):
        lat = hb.Lattice.from_description(line(k), device=0)
        work.copy_(c0)
        rec = lat.push_moments(work).cpu().numpy()[-1]
        lat.close()
        evals.append(1)
        return float(rec[6] + rec[17])                 # sigma_x^2 + sigma_y^2 at the end of the line

    start = np.array([1.0, 1.0])
    f0 = objective(start)
    res = minimize(objective, start, method="Nelder-Mead", options={"xatol": 1e-3, "fatol": 1e-12, "maxfev": 200})
    assert res.fun < 0.2 * f0 and len(evals) > 20          # the lenses really focus the beam
    ref, ref_rec = oracle.push(line(res.x), x)
    f_ref = ref_rec[-1][6] + ref_rec[-1][17]
    assert abs(res.fun - f_ref) <= 1e-4 * f_ref            # the GPU objective at the optimum is the oracle's
    for dk in ([0.3, 0.0], [0.0, -0.3]):                   # and it is a (local) minimum of the oracle's objective too
        _, r2 = oracle.push(line(res.x + np.array(dk)), x)
        assert r2[-1][6] + r2[-1][17] >= f_ref * (1 - 1e-6)


@pytest.mark.parametrize("run_mode", ["composed", "sequential"])
def test_set_element_rebuilds_only_its_run(hb, run_mode):
    """hb_lattice_set_element on a finalized lattice (P:68 'programmable at run time'): elements before and behind a
    COORD_T surrogate stage with energy gain (so the two runs have different reference momenta) are re-set, and the
    push must equal the oracle's push of the re-described lattice; the untouched lattice object is reused."""
    import torch
    desc, x = wl.config4(prec="fp32", n=30_000)
    els = desc["elements"]
    idx = [i for i, e in enumerate(els) if e["kind"] in ("quad", "drift", "sbend")]
    sur = [i for i, e in enumerate(els) if e["kind"] == "surrogate"]
    before = [i for i in idx if i < sur[0]] or [i for i in idx if i < sur[1]]
    behind = [i for i in idx if i > sur[-1]]
    assert before and behind
    lat = hb.Lattice.from_description(desc, run_mode=run_mode, device=0)
    c = hb.to_device(x)
    lat.push_moments(c)                                   # a push with the original elements first
    import copy
    new = copy.deepcopy(desc)
    for i, scale in ((before[0], 1.3), (behind[0], 0.7), (behind[-1], 1.1)):
        e = new["elements"][i]
        e["L"] = e["L"] * scale
        par = {"quad": "k", "sbend": "theta"}.get(e["kind"])
        if par:
            e[par] = e[par] * scale
        lat.set_element(i, e["L"], e[par] if par else 0.0)
    c = hb.to_device(x)
    rec = lat.push_moments(c).cpu().numpy()
    torch.cuda.synchronize()
    got = hb.to_host(c)
    lat.close()
    ref, ref_rec = oracle.push(new, x)
    err = np.max(np.abs(got.astype(np.float64) - ref), axis=1) / ref.std(axis=1)
    print("set_element", run_mode, "max err/std", err)
    assert err.max() <= 1e-5
    assert np.allclose(rec[-1][:6], np.asarray(ref_rec)[-1][:6], rtol=1e-4, atol=1e-9)
    old, _ = oracle.push(desc, x)
    assert (np.max(np.abs(old - ref), axis=1) / ref.std(axis=1)).max() > 1e-3     # the change was not a no-op


def test_stagewise_lens_optimisation_without_rebuilding(hb):
    """The paper's procedure on one cell: minimise eps_x behind a (synthetic) surrogate stage over the POSITION
    and STRENGTH of the plasma lens in front of it -- drift(d), lens(k), drift(D - d), stage, monitor.  One lattice is
    built once (weights packed and uploaded once); every Nelder-Mead evaluation is three hb_lattice_set_element calls
    and one hb_push_moments.  The optimum is checked with the fp64 oracle."""
    import torch
    from scipy.optimize import minimize
    widths = [6, 64, 64, 6]
    W, b = wl.make_mlp(widths, "xavier", 5, 0)
    x = wl.correlated_bunch(60_000, 41)
    f64 = x.astype(np.float64)
    sur = wl.surrogate(widths, W, b, "tanh", f64.mean(axis=1), f64.std(axis=1) * 3.0, f64.mean(axis=1), f64.std(axis=1),
                       prec="fp32")
    D, LL = 1.2, 0.05

    def line(v):
        d, k = float(v[0]), float(v[1])
        return wl.lattice([wl.drift(d), wl.plens(LL, k), wl.drift(D - d), sur, wl.monitor()])

    def eps_x(rec):
        return float(np.sqrt(max(rec[6] * rec[12] - rec[7] ** 2, 0.0)))

    lat = hb.Lattice.from_description(line([0.6, 1.0]), device=0)
    c0 = torch.from_numpy(x).cuda()
    work = torch.empty_like(c0)
    evals = []

    def objective(v):
        d = min(max(float(v[0]), 0.0), D)
        lat.set_element(0, d, 0.0)
        lat.set_element(1, LL, float(v[1]))
        lat.set_element(2, D - d, 0.0)
        work.copy_(c0)
        rec = lat.push_moments(work).cpu().numpy()[-1]
        evals.append(1)
        return eps_x(rec)

    start = np.array([0.6, 1.0])
    f0 = objective(start)
    res = minimize(objective, start, method="Nelder-Mead", options={"xatol": 1e-3, "fatol": 1e-13, "maxfev": 150})
    lat.close()
    assert len(evals) > 20 and res.fun <= f0
    v = np.array([min(max(res.x[0], 0.0), D), res.x[1]])
    _, ref_rec = oracle.push(line(v), x)
    f_ref = eps_x(np.asarray(ref_rec)[-1])
    print("stagewise optimisation:", len(evals), "evaluations, eps_x", f0, "->", res.fun, "oracle at optimum", f_ref)
    assert abs(res.fun - f_ref) <= 1e-3 * f_ref


def test_num_launches_counts_what_a_push_enqueues(hb):
    """hb_lattice_num_launches(n): one per run / stage (+ finalize per fused monitor, two per standalone monitor); a
    layered wide-net stage is one launch per linear layer and chunk of 2^20 particles"""
    desc, _ = wl.config1(prec="f16", n=8)
    lat = hb.Lattice.from_description(desc, device=0)
    assert lat.num_launches(False, 4096) == 3 and lat.num_launches(True, 4096) == 6 and lat.num_launches(True, 0) == 0
    lat.close()
    descp, _ = wl.paper_net(700, 3, prec="f16", particles=False)
    lat = hb.Lattice.from_description(descp, device=0)
    assert lat.num_launches(True, 10_000_000) == 10 * 4 + 1
    assert lat.num_launches(False, (1 << 20) + 1) == 2 * 4
    lat.close()
    lat = hb.Lattice.from_description(wl.lattice([wl.monitor(), wl.sbend(0.0, 0.0), wl.monitor()]), device=0)
    assert lat.num_launches(True, 100) == 2 + 2
    x = wl.gaussian_bunch(100, 3)
    c = hb.to_device(x)
    lat.push_moments(c)
    assert np.array_equal(hb.to_host(c), x)            # a zero-length, zero-angle bend is the identity
    lat.close()


# --------------------------------------------------------------------------------- NEXT-4: candidate settings in one pass
def test_push_candidates_against_the_oracle(hb):
    """hb_push_candidates: K settings (lens position and strength) of one transport gap over the same resident
    bunch; every record against the oracle, which pushes the bunch element by element through every candidate gap
    and takes the two-pass moments; and against the library's own push of that setting (which rounds to fp32)"""
    import torch
    gap = [wl.drift(0.3), wl.plens(0.05, 40.0), wl.drift(0.7), wl.quad(0.1, 1.2), wl.sbend(0.5, 0.02), wl.monitor()]
    desc = wl.lattice(gap, kinetic_MeV=8000.0)
    x = wl.gaussian_bunch(200_001, 61) + (wl.NOMINAL_SIGMA * [0.3, -0.2, 0.1, 0.4, 0.0, -0.5])[:, None].astype(np.float32)
    rng = np.random.default_rng(12)
    K = 37
    d0 = rng.uniform(0.05, 0.95, K)                       # lens position: drifts d0 and 1 - d0 around it
    kl = rng.uniform(-60.0, 80.0, K)                      # lens strength (both signs; one candidate without a lens)
    kl[5] = 0.0
    length = np.stack([d0, np.full(K, 0.05), 1.0 - d0], axis=1)
    param = np.stack([np.zeros(K), kl, np.zeros(K)], axis=1)
    lat = hb.Lattice.from_description(desc, device=0)
    c = hb.to_device(x)
    rec = lat.push_candidates(c, [0, 1, 2], length, param).cpu().numpy()
    assert np.array_equal(hb.to_host(c), x)               # the bunch is only read
    assert rec.shape == (K, 27) and np.all(np.isfinite(rec))
    worst = 0.0
    for k in range(K):
        dk = wl.lattice([wl.drift(d0[k]), wl.plens(0.05, kl[k]), wl.drift(1.0 - d0[k])] + gap[3:], kinetic_MeV=8000.0)
        _, ref = oracle.push(dk, x)
        R = sym(ref[0]); C = sym(rec[k]); sd = np.sqrt(np.diag(R))
        worst = max(worst, np.max(np.abs(rec[k][:6] - ref[0][:6]) / sd), np.max(np.abs(C - R) / np.outer(sd, sd)))
    print("candidates vs oracle: worst moment error / (sigma_j sigma_k):", worst)
    assert worst <= 1e-9
    # the same setting through set_element + push_moments (fp32 images): 1e-6
    for k in (0, 5, 36):
        for j in range(3):
            lat.set_element(j, length[k, j], param[k, j])
        c2 = hb.to_device(x)
        r2 = lat.push_moments(c2).cpu().numpy()[0]
        moments_close(rec[k], r2, 1e-6)
    # the lattice was not changed by the candidates call, K = 0 and n = 0 are legal
    assert lat.push_candidates(c, [1], np.zeros((0, 1)), np.zeros((0, 1))).shape == (0, 27)
    e = torch.zeros((6, 0), dtype=torch.float32, device="cuda")
    assert bool(torch.isnan(lat.push_candidates(e, [1], [[0.05]], [[1.0]])).all())
    lat.close()


def test_push_candidates_errors(hb):
    W, b = wl.make_mlp([6, 8, 6], "xavier", 1, 0)
    z, o = np.zeros(6), np.ones(6)
    desc = wl.lattice([wl.drift(0.5), wl.quad(0.1, 1.0), wl.surrogate([6, 8, 6], W, b, "tanh", z, o, z, o),
                       wl.drift(0.5), wl.drift_exact(0.2), wl.monitor()])
    lat = hb.Lattice.from_description(desc, device=0)
    c = hb.to_device(wl.gaussian_bunch(1000, 3))
    for idx, L, p in (([0, 3], [[0.1, 0.1]], [[0, 0]]),          # two different runs
                      ([2], [[0.1]], [[0.0]]),                   # a surrogate stage
                      ([1], [[-0.1]], [[1.0]]),                  # negative quadrupole length
                      ([1], [[0.1]], [[float("nan")]])):
        with pytest.raises(hb.HbError) as e:
            lat.push_candidates(c, idx, L, p)
        assert e.value.status == 1
    with pytest.raises(hb.HbError) as e:                       # the second run holds an exact drift: no composed map
        lat.push_candidates(c, [3], [[0.1]], [[0.0]])
    assert e.value.status == 5
    lat.close()
