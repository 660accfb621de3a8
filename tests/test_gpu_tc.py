"""Tensor-core surrogate (tcgen05) vs the fp64 oracle, through the C ABI (-m gpu).

BASELINE.json asks <= 2e-2 x std(oracle's output coordinate) for the 16-bit path.  DESIGN.md 6.5 records what is
measured: HB_PREC_F16 (and tf32) meet it; plain bf16 operands (8 significand bits) do not on the random synthetic nets.
Plain bf16 is therefore NOT a conforming mode: its entries below are regression bounds at the largest error on record
(1.1e-1, C3 at N = 1e7), and tests/test_gpu_stagefed.py::test_plain_bf16_does_not_meet_the_north_star_bound states the
miss against 2e-2 itself (strict xfail).
"""
import os

import numpy as np
import pytest

import oracle
import workloads as wl

pytestmark = pytest.mark.gpu

TOL = {"f16": 2e-2, "bf16": 1.2e-1}


@pytest.fixture(scope="module")
def hb():
    import torch
    assert torch.cuda.is_available()
    import paper_2402_17248_b200 as hb
    hb.lib()
    return hb


def gpu_push(hb, desc, x, moments=False, prec=None):
    import torch
    lat = hb.Lattice.from_description(desc, device=0, prec=prec)
    c = hb.to_device(x)
    rec = lat.push_moments(c) if moments else lat.push(c)
    torch.cuda.synchronize()
    out = hb.to_host(c).astype(np.float64)
    lat.close()
    return out, (None if rec is None else rec.cpu().numpy())


def rel_err(got, ref):
    return np.max(np.abs(got - ref), axis=1) / ref.std(axis=1)


def identity_net(H, prec):
    A0 = np.zeros((H, 6), np.float32); A0[:6] = np.eye(6)
    A1 = np.zeros((H, H), np.float32); A1[:6, :6] = np.eye(6)
    A2 = np.zeros((6, H), np.float32); A2[:, :6] = np.eye(6)
    zb = [np.zeros(H, np.float32), np.zeros(H, np.float32), np.zeros(6, np.float32)]
    z, o = np.zeros(6), np.ones(6)
    return wl.surrogate([6, H, H, 6], [A0, A1, A2], zb, "prelu", z, o, z, o, prelu_a=[1.0, 1.0], prec=prec)


@pytest.mark.parametrize("force_cg", ["1", "2"])
@pytest.mark.parametrize("prec", ["bf16", "f16"])
def test_tc_bringup_identity_net(hb, prec, force_cg, monkeypatch):
    """one tile, identity weights: output = input rounded to the operand type (descriptor / layout check)"""
    if force_cg == "2":
        monkeypatch.setenv("HB_TC_FORCE_CG", "2")
    else:
        monkeypatch.delenv("HB_TC_FORCE_CG", raising=False)
    x = wl.gaussian_bunch(128, 3, sigma=np.ones(6))
    got, _ = gpu_push(hb, wl.lattice([identity_net(64, prec)]), x)
    eps = 2.0 ** -8 if prec == "bf16" else 2.0 ** -11
    assert np.all(np.isfinite(got))
    assert np.max(np.abs(got - x) / np.maximum(np.abs(x), 1e-3)) <= 1.01 * eps


@pytest.mark.parametrize("force_cg", ["1", "2"])
@pytest.mark.parametrize("n", [1, 127, 128, 129, 300, 5000, 40_001])
def test_tc_tiles_and_tails(hb, n, force_cg, monkeypatch):
    if force_cg == "2":
        monkeypatch.setenv("HB_TC_FORCE_CG", "2")
    else:
        monkeypatch.delenv("HB_TC_FORCE_CG", raising=False)
    desc, _ = wl.config1(prec="f16", n=8)
    desc = wl.lattice(desc["elements"][6:8])          # surrogate + monitor
    x = wl.gaussian_bunch(max(n, 8), 17)[:, :n].copy()
    ref, ref_rec = oracle.push(desc, x)
    got, rec = gpu_push(hb, desc, x, moments=True)
    assert np.all(np.isfinite(got))
    # G14: std of the oracle's output coordinate -- over 5000 particles of the same generator (n itself may be 1)
    big, _ = oracle.push(desc, wl.gaussian_bunch(5000, 17))
    assert np.max(np.abs(got - ref) / big.std(axis=1)[:, None]) <= 2e-2
    own = oracle.moments(np.ascontiguousarray(got))
    assert np.allclose(rec[0][:6], own[:6], rtol=1e-9, atol=1e-16)
    if n > 1:
        assert np.allclose(rec[0][6:], own[6:], rtol=1e-7, atol=1e-20)


@pytest.mark.parametrize("prec", ["bf16", "f16"])
def test_config1_tensor_core(hb, prec):
    desc, x = wl.config1(prec=prec)
    ref, ref_rec = oracle.push(desc, x)
    got, rec = gpu_push(hb, desc, x, moments=True)
    e = rel_err(got, ref)
    print("C1", prec, "err/std:", e)
    assert e.max() <= TOL[prec]


@pytest.mark.parametrize("one_tile", ["0", "1"])
@pytest.mark.parametrize("prec", ["bf16", "f16"])
@pytest.mark.parametrize("act,widths", [("relu", [6, 64, 6]), ("tanh", [6, 128, 128, 128, 6]),
                                        ("prelu", [6, 100, 37, 6]), ("relu", [6, 256, 256, 256, 6]),
                                        ("identity", [6, 192, 6]), ("tanh", [6, 256, 256, 6])])
def test_tc_shapes(hb, prec, act, widths, one_tile, monkeypatch):
    """resident-weights kernels vs the oracle.  Nets wider than 128 run on the two-tiles-in-flight kernel
    (hb_sur_tc2.cu) unless HB_TC_ONE_TILE=1 (read at finalize) keeps them on the one-tile kernel (hb_sur_tc.cu)"""
    if one_tile == "1":
        if max(widths[1:-1]) <= 128:
            pytest.skip("narrow nets run on the one-tile kernel anyway")
        monkeypatch.setenv("HB_TC_ONE_TILE", "1")
    else:
        monkeypatch.delenv("HB_TC_ONE_TILE", raising=False)
    n = 20_000
    init = "he" if act in ("relu", "prelu") else "xavier"
    W, b = wl.make_mlp(widths, init, 55, len(widths))
    rng = np.random.default_rng(6)
    a = rng.uniform(0.05, 0.3, len(widths) - 2).astype(np.float32) if act == "prelu" else None
    x = wl.correlated_bunch(n, 41)
    x64 = x.astype(np.float64)
    sur = wl.surrogate(widths, W, b, act, x64.mean(axis=1), x64.std(axis=1), rng.normal(size=6),
                       rng.uniform(0.5, 2.0, 6), prelu_a=a, prec=prec)
    desc = wl.lattice([sur, wl.monitor()])
    ref, ref_rec = oracle.push(desc, x)
    got, rec = gpu_push(hb, desc, x, moments=True)
    e = rel_err(got, ref)
    rms = np.sqrt(np.mean((got - ref) ** 2, axis=1)) / ref.std(axis=1)
    print("shape", widths, act, prec, "max err/std", e.max(), "rms err/std", rms.max())
    assert np.all(np.isfinite(got))
    assert e.max() <= TOL[prec]


@pytest.mark.parametrize("prec", ["bf16", "f16"])
def test_config4_tensor_core_per_stage(hb, prec):
    """COORD_T stage (s<->t in deviation form fused) on tensor cores; stage fed with the oracle's state."""
    desc, x = wl.config4(prec=prec, n=50_000, stages=2)
    d1 = wl.lattice(desc["elements"][:1])
    r1, _ = oracle.push(d1, x)
    g1, _ = gpu_push(hb, d1, x)
    e1 = rel_err(g1, r1)
    print("C4 stage 1", prec, "err/std:", e1)
    assert np.all(np.isfinite(g1)) and e1.max() <= TOL[prec]
    ref, ref_rec = oracle.push(desc, x)
    got, rec = gpu_push(hb, desc, x, moments=True)
    e = rel_err(got, ref)
    print("C4 free-running 2 stages", prec, "err/std:", e)
    assert np.all(np.isfinite(got))
    # (every stage fed from the oracle, incl. stage 2 with its 8 GeV reference: tests/test_gpu_stagefed.py)


# ------------------------------------------------------------------ streamed-weights kernel (hb_sur_tcs.cu)
@pytest.mark.parametrize("prec", ["bf16", "f16"])
@pytest.mark.parametrize("H", [128, 512])
def test_tcs_bringup_identity_net(hb, prec, H, monkeypatch):
    """identity weights through the streamed kernel: ring blocks, N halves, descriptors, A_FREE protocol"""
    monkeypatch.setenv("HB_TC_FORCE_STREAM", "1")
    x = wl.gaussian_bunch(3000, 3, sigma=np.ones(6))
    got, _ = gpu_push(hb, wl.lattice([identity_net(H, prec)]), x)
    eps = 2.0 ** -8 if prec == "bf16" else 2.0 ** -11
    assert np.all(np.isfinite(got))
    assert np.max(np.abs(got - x) / np.maximum(np.abs(x), 1e-3)) <= 1.01 * eps


@pytest.mark.parametrize("prec", ["bf16", "f16"])
@pytest.mark.parametrize("act,widths", [("relu", [6, 256, 256, 256, 6]), ("tanh", [6, 128, 128, 128, 6]),
                                        ("tanh", [6, 512, 512, 512, 512, 6]), ("prelu", [6, 300, 300, 6]),
                                        ("relu", [6, 500, 6]), ("identity", [6, 384, 384, 384, 384, 384, 6])])
def test_tcs_shapes(hb, prec, act, widths, monkeypatch):
    """streamed kernel vs the oracle (forced for shapes the resident kernel would take)"""
    monkeypatch.setenv("HB_TC_FORCE_STREAM", "1")
    n = 20_000
    init = "he" if act in ("relu", "prelu") else "xavier"
    W, b = wl.make_mlp(widths, init, 56, len(widths))
    rng = np.random.default_rng(7)
    a = rng.uniform(0.05, 0.3, len(widths) - 2).astype(np.float32) if act == "prelu" else None
    x = wl.correlated_bunch(n, 42)
    x64 = x.astype(np.float64)
    sur = wl.surrogate(widths, W, b, act, x64.mean(axis=1), x64.std(axis=1), rng.normal(size=6),
                       rng.uniform(0.5, 2.0, 6), prelu_a=a, prec=prec)
    desc = wl.lattice([sur, wl.monitor()])
    ref, ref_rec = oracle.push(desc, x)
    got, rec = gpu_push(hb, desc, x, moments=True)
    e = rel_err(got, ref)
    rms = np.sqrt(np.mean((got - ref) ** 2, axis=1)) / ref.std(axis=1)
    print("streamed shape", widths, act, prec, "max err/std", e.max(), "rms err/std", rms.max())
    assert np.all(np.isfinite(got))
    assert e.max() <= TOL[prec]
    own = oracle.moments(np.ascontiguousarray(got))
    assert np.allclose(rec[0][:6], own[:6], rtol=1e-9, atol=1e-16)


@pytest.mark.parametrize("n", [1, 129, 257, 40_001])
def test_tcs_tiles_and_tails(hb, n, monkeypatch):
    monkeypatch.setenv("HB_TC_FORCE_STREAM", "1")
    widths = [6, 128, 128, 6]
    W, b = wl.make_mlp(widths, "xavier", 57, 3)
    z, o = np.zeros(6), np.ones(6)
    x = wl.gaussian_bunch(max(n, 8), 18, sigma=np.ones(6))[:, :n].copy()
    desc = wl.lattice([wl.surrogate(widths, W, b, "tanh", z, o, z, o, prec="f16"), wl.monitor()])
    ref, _ = oracle.push(desc, x)
    got, rec = gpu_push(hb, desc, x, moments=True)
    assert np.all(np.isfinite(got))
    assert np.max(np.abs(got - ref)) <= 2e-2
    own = oracle.moments(np.ascontiguousarray(got))
    assert np.allclose(rec[0][:6], own[:6], rtol=1e-9, atol=1e-16)


# ------------------------------------------------------------------ two tiles in flight, N-halves (hb_sur_tc2.cu)
@pytest.mark.parametrize("force_cg", ["1", "2"])
@pytest.mark.parametrize("prec", ["bf16", "f16"])
def test_tc2_bringup_identity_net(hb, prec, force_cg, monkeypatch):
    """identity weights, H = 256: output = input rounded to the operand type (half-N weight rows, operand columns,
    descriptors of both cluster sizes)"""
    monkeypatch.delenv("HB_TC_ONE_TILE", raising=False)
    if force_cg == "2":
        monkeypatch.setenv("HB_TC_FORCE_CG", "2")
    else:
        monkeypatch.delenv("HB_TC_FORCE_CG", raising=False)
    x = wl.gaussian_bunch(3000, 3, sigma=np.ones(6))
    got, _ = gpu_push(hb, wl.lattice([identity_net(256, prec)]), x)
    eps = 2.0 ** -8 if prec == "bf16" else 2.0 ** -11
    assert np.all(np.isfinite(got))
    assert np.max(np.abs(got - x) / np.maximum(np.abs(x), 1e-3)) <= 1.01 * eps


@pytest.mark.parametrize("force_cg", ["1", "2"])
@pytest.mark.parametrize("prec", ["bf16", "f16"])
@pytest.mark.parametrize("act,widths,n", [("relu", [6, 256, 256, 256, 6], 70_000), ("tanh", [6, 192, 192, 6], 20_001),
                                          ("prelu", [6, 130, 250, 140, 6], 333), ("relu", [6, 160, 6], 40_001),
                                          ("tanh", [6, 256, 6], 1), ("identity", [6, 200, 256, 6], 257),
                                          ("prelu", [6, 256, 64, 256, 6], 129), ("relu", [6, 16, 256, 256, 256, 6], 5_000)])
def test_tc2_shapes(hb, prec, act, widths, n, force_cg, monkeypatch):
    """two-tile kernel vs the oracle: odd numbers of tile groups per CTA (slot 1 one tile short), ragged tails, one
    hidden layer (phases a, d only), unequal widths (N-halves of 96 / 128 / 32 columns), a narrow first layer,
    single CTAs and CTA pairs; moments"""
    monkeypatch.delenv("HB_TC_ONE_TILE", raising=False)
    if force_cg == "2":
        monkeypatch.setenv("HB_TC_FORCE_CG", "2")
    else:
        monkeypatch.delenv("HB_TC_FORCE_CG", raising=False)
    init = "he" if act in ("relu", "prelu") else "xavier"
    W, b = wl.make_mlp(widths, init, 58, len(widths))
    rng = np.random.default_rng(8)
    a = rng.uniform(0.05, 0.3, len(widths) - 2).astype(np.float32) if act == "prelu" else None
    full = wl.correlated_bunch(max(n, 2000), 43)
    x = full[:, :n].copy()
    f64 = full.astype(np.float64)
    sur = wl.surrogate(widths, W, b, act, f64.mean(axis=1), f64.std(axis=1), rng.normal(size=6),
                       rng.uniform(0.5, 2.0, 6), prelu_a=a, prec=prec)
    desc = wl.lattice([sur, wl.monitor()])
    ref, _ = oracle.push(desc, x)
    got, rec = gpu_push(hb, desc, x, moments=True)
    big = ref if n >= 1000 else oracle.push(desc, full[:, :2000])[0]
    e = np.max(np.abs(got - ref), axis=1) / big.std(axis=1)          # G14 (2000 particles of the same bunch when n is tiny)
    print("two-tile shape", widths, act, prec, "cg", force_cg, "max err/std", e.max())
    assert np.all(np.isfinite(got))
    assert e.max() <= TOL[prec]
    own = oracle.moments(np.ascontiguousarray(got))
    assert np.allclose(rec[0][:6], own[:6], rtol=1e-9, atol=1e-16)


# ------------------------------------------------------------------ HB_PREC_TF32 (kind::tf32 on the streamed kernel)
def test_tf32_bringup_identity_net(hb):
    """identity weights, tf32 operands: output = input rounded to 10 explicit mantissa bits (layouts, descriptors)"""
    x = wl.gaussian_bunch(3000, 3, sigma=np.ones(6))
    got, _ = gpu_push(hb, wl.lattice([identity_net(128, "tf32")]), x)
    assert np.all(np.isfinite(got))
    assert np.max(np.abs(got - x) / np.maximum(np.abs(x), 1e-3)) <= 1.01 * 2.0 ** -11


@pytest.mark.parametrize("act,widths,n", [("relu", [6, 256, 256, 256, 6], 20_000), ("tanh", [6, 128, 128, 128, 6], 20_000),
                                          ("prelu", [6, 100, 100, 6], 257), ("tanh", [6, 192, 6], 1),
                                          ("identity", [6, 64, 64, 64, 64, 64, 6], 40_001)])
def test_tf32_shapes(hb, act, widths, n):
    init = "he" if act in ("relu", "prelu") else "xavier"
    W, b = wl.make_mlp(widths, init, 59, len(widths))
    rng = np.random.default_rng(9)
    a = rng.uniform(0.05, 0.3, len(widths) - 2).astype(np.float32) if act == "prelu" else None
    x = wl.correlated_bunch(max(n, 8), 44)[:, :n].copy()
    full = wl.correlated_bunch(max(n, 8), 44).astype(np.float64)
    sur = wl.surrogate(widths, W, b, act, full.mean(axis=1), full.std(axis=1), rng.normal(size=6),
                       rng.uniform(0.5, 2.0, 6), prelu_a=a, prec="tf32")
    desc = wl.lattice([sur, wl.monitor()])
    ref, _ = oracle.push(desc, x)
    got, rec = gpu_push(hb, desc, x, moments=True)
    # G14: std of the oracle's output coordinate (over 5000 particles of the same generator when n is tiny)
    big, _ = oracle.push(desc, wl.correlated_bunch(5000, 44))
    scale = ref.std(axis=1) if n >= 1000 else big.std(axis=1)
    e = np.max(np.abs(got - ref), axis=1) / scale
    print("tf32 shape", widths, act, "max err/std", e.max())
    assert np.all(np.isfinite(got))
    assert e.max() <= 2e-2
    own = oracle.moments(np.ascontiguousarray(got))
    assert np.allclose(rec[0][:6], own[:6], rtol=1e-9, atol=1e-16)


def test_tf32_unsupported_shapes_fail_loudly(hb):
    """tf32 needs the streamed kernel's shape (equal hidden widths <= 256); anything else is an error, never a fallback"""
    W, b = wl.make_mlp([6, 512, 512, 6], "xavier", 60, 3)
    z, o = np.zeros(6), np.ones(6)
    with pytest.raises(Exception):
        hb.Lattice.from_description(wl.lattice([wl.surrogate([6, 512, 512, 6], W, b, "tanh", z, o, z, o, prec="tf32")]), device=0)


# ------------------------------------------------------------------ wide nets: one launch per layer (hb_sur_tcw.cu)
@pytest.mark.parametrize("prec", ["bf16", "f16"])
@pytest.mark.parametrize("H", [768, 1024])
def test_tcw_bringup_identity_net(hb, prec, H):
    """identity weights through the layered kernel: pre-tiled scratch, ring stages, output blocks, bulk stores"""
    x = wl.gaussian_bunch(3000, 3, sigma=np.ones(6))
    got, _ = gpu_push(hb, wl.lattice([identity_net(H, prec)]), x)
    eps = 2.0 ** -8 if prec == "bf16" else 2.0 ** -11
    assert np.all(np.isfinite(got))
    assert np.max(np.abs(got - x) / np.maximum(np.abs(x), 1e-3)) <= 1.01 * eps


@pytest.mark.parametrize("prec", ["bf16", "f16"])
@pytest.mark.parametrize("act,widths,n", [("prelu", [6, 900, 900, 900, 900, 900, 6], 20_000), ("prelu", [6, 700, 700, 700, 6], 20_000),
                                          ("tanh", [6, 520, 520, 6], 257), ("relu", [6, 1024, 6], 1),
                                          ("relu", [6, 600, 600, 6], 40_001), ("tanh", [6, 900, 930, 960, 6], 3_000)])
def test_tcw_shapes(hb, prec, act, widths, n):
    """the paper's own network shapes (6-900^5-6, 6-700^3-6 PReLU) and the edges of the layered kernel"""
    init = "he" if act in ("relu", "prelu") else "xavier"
    W, b = wl.make_mlp(widths, init, 61, len(widths))
    rng = np.random.default_rng(10)
    a = rng.uniform(0.05, 0.3, len(widths) - 2).astype(np.float32) if act == "prelu" else None
    full = wl.correlated_bunch(max(n, 8), 45)
    x = full[:, :n].copy()
    f64 = full.astype(np.float64)
    sur = wl.surrogate(widths, W, b, act, f64.mean(axis=1), f64.std(axis=1), rng.normal(size=6),
                       rng.uniform(0.5, 2.0, 6), prelu_a=a, prec=prec)
    desc = wl.lattice([sur, wl.monitor()])
    assert hb.hb_surrogate_kernel(prec, widths) == "tcgen05-layered"
    ref, _ = oracle.push(desc, x)
    got, rec = gpu_push(hb, desc, x, moments=True)
    big, _ = oracle.push(desc, wl.correlated_bunch(2000, 45)) if n < 1000 else (ref, None)
    scale = big.std(axis=1)                            # G14 (over 2000 particles of the same bunch when n is tiny)
    e = np.max(np.abs(got - ref), axis=1) / scale
    print("layered shape", widths, act, prec, "max err/std", e.max())
    assert np.all(np.isfinite(got))
    assert e.max() <= TOL[prec]
    own = oracle.moments(np.ascontiguousarray(got))
    assert np.allclose(rec[0][:6], own[:6], rtol=1e-9, atol=1e-16)
