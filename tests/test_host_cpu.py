"""CPU-only checks of the boundary: the library loads, exports every symbol of include/hb.h,
validates arguments on the host, and fails loudly (never falls back) without a device."""
import os
import re

import numpy as np
import pytest

import workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def hb():
    from paper_2402_17248_b200.build import build_lib
    build_lib()
    import paper_2402_17248_b200 as hb
    hb.lib()
    return hb


def test_every_declared_symbol_is_exported(hb):
    hdr = open(os.path.join(ROOT, "include", "hb.h")).read()
    declared = set(re.findall(r"\b(hb_[a-z0-9_]+)\s*\(", hdr))
    assert declared, "no declarations parsed"
    assert declared == set(hb.EXPORTED_SYMBOLS)
    L = hb.lib()
    for name in declared:
        assert getattr(L, name) is not None


def test_host_validation_without_device(hb):
    assert hb.hb_status_string(0) == "HB_OK" and hb.hb_status_string(5) == "HB_ERR_UNSUPPORTED"
    with pytest.raises(hb.HbError) as e:
        hb.hb_lattice_create(float("nan"), 0.511)
    assert e.value.status == 1
    h = hb.hb_lattice_create(1000.0, wl.ELECTRON_MEV)
    hb.hb_lattice_add_element(h, "drift", -0.5)                 # negative drift length is legal
    hb.hb_lattice_add_element(h, "monitor")
    with pytest.raises(hb.HbError):
        hb.hb_lattice_add_element(h, "sbend", -0.5, 0.01)
    with pytest.raises(hb.HbError):
        hb.hb_lattice_add_element(h, "quad", 0.1, float("inf"))
    with pytest.raises(hb.HbError) as e:                        # zero-length bend with an angle: infinite curvature
        hb.hb_lattice_add_element(h, "sbend", 0.0, 0.02)
    assert e.value.status == 1
    hb.hb_lattice_add_element(h, "sbend", 0.0, 0.0)             # ... without an angle it is the identity
    with pytest.raises(hb.HbError) as e:
        hb.hb_lattice_set_element(h, 2, 0.0, 0.02)
    assert e.value.status == 1
    with pytest.raises(hb.HbError) as e:
        hb.hb_lattice_set_centroid(h, [0, 0, float("nan"), 0, 0, 0])
    assert e.value.status == 1
    hb.hb_lattice_set_centroid(h, [1e-3, 0, 0, 0, 0, 0])
    W, b = wl.make_mlp([6, 8, 6], "xavier", 1, 0)
    z, o = np.zeros(6), np.ones(6)
    hb.hb_lattice_add_surrogate(h, [6, 8, 6], W, b, "tanh", z, o, z, o)
    with pytest.raises(hb.HbError):
        hb.hb_lattice_add_surrogate(h, [6, 8, 6], W, b, "tanh", z, np.array([1, 1, 0, 1, 1, 1.0]), z, o)
    with pytest.raises(hb.HbError):
        hb.hb_lattice_add_surrogate(h, [6, 8, 6], W, b, "prelu", z, o, z, o)      # slopes missing
    assert hb.hb_lattice_num_monitors(h) == 1
    hb.hb_lattice_destroy(h)


def test_no_cpu_fallback(hb):
    import torch
    if torch.cuda.is_available():
        pytest.skip("device present")
    h = hb.hb_lattice_create(1000.0, wl.ELECTRON_MEV)
    hb.hb_lattice_add_element(h, "drift", 1.0)
    with pytest.raises(hb.HbError) as e:
        hb.hb_lattice_finalize(h, 0)
    assert e.value.status in (4, 5)
    with pytest.raises(hb.HbError) as e:
        hb.hb_push(h, 0, 0, 0, 0, 0, 0, 0, 0)
    assert e.value.status == 2
    hb.hb_lattice_destroy(h)


def test_product_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_2402_17248_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.replace("the oracle", "").replace("oracle/", "").replace("by the oracle", ""), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2402_17248_b200" not in src and "libhb" not in src


def test_shard_ranges_cover_everything():
    for n in (0, 1, 7, 10_000_001):
        for w in (1, 2, 3, 8):
            r = [wl.shard_range(n, k, w) for k in range(w)]
            assert r[0][0] == 0 and r[-1][1] == n
            assert all(a[1] == b[0] for a, b in zip(r[:-1], r[1:]))
            assert max(b - a for a, b in r) - min(b - a for a, b in r) <= 1


def test_surrogate_kernel_dispatch_is_a_host_decision(hb, monkeypatch):
    """which kernel a shape runs on (the decision hb_lattice_finalize takes) -- BASELINE.json's five configs and the
    edges of each kernel's envelope; unsupported shapes are an error with a reason, never a fallback"""
    for k in ("HB_TC_FORCE_STREAM", "HB_TC_FORCE_CG", "HB_TC_OCC2", "HB_TC_ONE_TILE"):
        monkeypatch.delenv(k, raising=False)
    K = hb.hb_surrogate_kernel
    assert K("fp32", [6, 64, 64, 6]) == "fp32-ffma"                       # C1 as specified
    assert K("bf16", [6, 64, 64, 6]) == "tcgen05-resident"
    assert K("bf16", [6, 256, 256, 256, 6]) == "tcgen05-resident"         # C3: 272 KB of weights over a CTA pair
    assert K("f16", [6, 128, 128, 128, 6]) == "tcgen05-resident"          # C4
    assert K("bf16", [6, 512, 512, 512, 512, 6]) == "tcgen05-streamed"    # C5: 1.55 MB of weights
    assert K("bf16", [6] + [256] * 8 + [6]) == "tcgen05-streamed"         # too deep to stay resident
    assert K("bf16", [6, 6]) == "tcgen05-resident"                        # no hidden layer
    assert K("tf32", [6, 256, 256, 256, 6]) == "tcgen05-streamed"
    assert K("tf32", [6, 512, 512, 6]) is None and "TF32" in hb.hb_last_error()
    assert K("bf16", [6, 900, 900, 900, 900, 900, 6]) == "tcgen05-layered"   # the paper's own nets: one launch per layer
    assert K("f16", [6, 700, 700, 700, 6]) == "tcgen05-layered"
    assert K("tf32", [6, 700, 700, 700, 6]) is None and K("bf16", [6, 1100, 1100, 6]) is None
    assert K("bf16", [6, 900, 930, 960, 6]) == "tcgen05-layered"          # unequal widths that pad to the same multiple of 64
    assert K("bf16", [6, 512, 300, 512, 6]) is None
    assert K("bf16", [6, 512, 1024, 512, 6]) is None                      # streamed / layered kernels: equal padded widths only
    assert K("bf16", [6, 1025, 6]) is None and K("bf16", [5, 8, 6]) is None
    monkeypatch.setenv("HB_TC_FORCE_STREAM", "1")
    assert K("bf16", [6, 256, 256, 256, 6]) == "tcgen05-streamed"


def test_moments_merge_against_plain_moments(hb):
    """hb_moments_merge (host arithmetic of the sharded monitor): records of parts -> record of the whole, against
    numpy's mean / covariance of the concatenation; uneven three-way split, far-off-centre data, empty parts,
    aliasing, NULL"""
    rng = np.random.default_rng(5)
    a = rng.normal(size=(6, 1000)) * np.array([1e-3, 1e-4, 2e-3, 1e-4, 5e-4, 1e-3])[:, None] + 0.25
    a[1] += 3.0 * a[0]                                  # off-diagonal terms that matter

    def rec(z):
        m = z.mean(axis=1)
        c = np.cov(z, bias=True)
        return np.concatenate([m, c[np.triu_indices(6)]])

    cuts = [0, 17, 640, 1000]
    acc, n_acc = None, 0
    for lo, hi in zip(cuts[:-1], cuts[1:]):
        r = rec(a[:, lo:hi])
        acc = r if acc is None else hb.hb_moments_merge(acc, n_acc, r, hi - lo)
        n_acc += hi - lo
    want = rec(a)
    assert np.allclose(acc[:6], want[:6], rtol=1e-14)
    scale = np.sqrt(np.outer(np.diag(np.cov(a, bias=True)), np.diag(np.cov(a, bias=True))))[np.triu_indices(6)]
    assert np.all(np.abs(acc[6:] - want[6:]) <= 1e-9 * scale)   # 0.25 offset: cancellation costs a few digits
    nan = np.full(27, np.nan)
    assert np.array_equal(hb.hb_moments_merge(nan, 0, want, 1000), want)
    assert np.array_equal(hb.hb_moments_merge(want, 1000, nan, 0), want)
    assert np.all(np.isnan(hb.hb_moments_merge(nan, 0, nan, 0)))
    # two single particles: mean = midpoint, C = d d^T / 4
    p, q = a[:, 0], a[:, 1]
    z = np.zeros(21)
    got = hb.hb_moments_merge(np.concatenate([p, z]), 1, np.concatenate([q, z]), 1)
    d = q - p
    assert np.allclose(got[:6], 0.5 * (p + q), rtol=1e-15)
    assert np.allclose(got[6:], (np.outer(d, d) / 4)[np.triu_indices(6)], rtol=1e-12, atol=0)
    import ctypes
    assert hb.lib().hb_moments_merge(None, 1, None, 1, None) != 0
    out = want.copy()
    pd = ctypes.POINTER(ctypes.c_double)
    r2 = rec(a[:, :500])
    exp = hb.hb_moments_merge(out, 1000, r2, 500)
    assert hb.lib().hb_moments_merge(out.ctypes.data_as(pd), 1000, r2.ctypes.data_as(pd), 500, out.ctypes.data_as(pd)) == 0
    assert np.array_equal(out, exp)


def test_set_element_host_validation(hb):
    """hb_lattice_set_element before finalize is pure host logic: index and value checks, kinds that cannot be re-set"""
    lat = hb.hb_lattice_create(1000.0, wl.ELECTRON_MEV)
    hb.hb_lattice_add_element(lat, "drift", 1.0)
    hb.hb_lattice_add_element(lat, "quad", 0.3, 2.0)
    hb.hb_lattice_add_element(lat, "monitor")
    hb.hb_lattice_add_multipole(lat, 3, 0.5, 0.0)
    hb.hb_lattice_set_element(lat, 0, -0.5)              # negative drift length is allowed (as in add_element)
    hb.hb_lattice_set_element(lat, 1, 0.2, -3.0)
    for args in ((4, 1.0, 0.0), (-1, 1.0, 0.0), (2, 1.0, 0.0), (3, 1.0, 0.0), (1, -0.1, 1.0), (1, 0.1, float("nan")),
                 (0, float("inf"), 0.0)):
        with pytest.raises(hb.HbError) as e:
            hb.hb_lattice_set_element(lat, *args)
        assert e.value.status == 1                       # HB_ERR_INVALID_ARG
    hb.hb_lattice_destroy(lat)


def test_profile_traffic_table_names_existing_captures():
    """bench.py reads roofline.traffic from profiles/ncu_traffic.json: every capture it names is committed"""
    import json
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    with open(os.path.join(root, "profiles", "ncu_traffic.json")) as f:
        table = json.load(f)
    assert table["entries"]
    for e in table["entries"]:
        assert os.path.exists(os.path.join(root, "profiles", e["capture"])), e["capture"]
        assert e["dram_bytes"] > 0 and e["n"] > 0 and e["kernel"].startswith("hb_")
