"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (-m gpu).

Every step of the path is a per-particle map, so the fp64 oracle can compute any particle of a 1e7 / 1e8
bunch on its own: the GPU pushes the whole bunch through the C ABI, the oracle pushes a seeded sample of it
(first tile, last tile, ragged tail, and a spread of particles in between), and the two are compared element by
element.  The moment records are checked by a property that holds at any size: the record the kernels reduce on
the device equals the plain fp64 moments (oracle R10) of the very output they wrote.
"""
import numpy as np
import pytest

import oracle
import workloads as wl

pytestmark = pytest.mark.gpu

TOL = {"f16": 2e-2, "bf16": 1.2e-1, "fp32": 1e-5}      # bf16: regression bound at the measured level (test_gpu_tc.py)


@pytest.fixture(scope="module")
def hb():
    import torch
    assert torch.cuda.is_available()
    import paper_2402_17248_b200 as hb
    hb.lib()
    return hb


def sample_indices(n, m=6000, seed=99):
    rng = np.random.default_rng(seed)
    edge = np.concatenate([np.arange(0, min(n, 300)), np.arange(max(0, n - 300), n)])
    mid = rng.integers(0, n, size=m)
    return np.unique(np.concatenate([edge, mid]))


def gpu_push_full(hb, desc, x, prec=None):
    import torch
    lat = hb.Lattice.from_description(desc, device=0, prec=prec)
    c = hb.to_device(x)
    rec = lat.push_moments(c)
    torch.cuda.synchronize()
    out = hb.to_host(c)
    lat.close()
    del c
    torch.cuda.empty_cache()
    return out, rec.cpu().numpy()


def check_moments(rec_last, out):
    own = oracle.moments(np.ascontiguousarray(out.astype(np.float64)))
    assert np.allclose(rec_last[:6], own[:6], rtol=1e-9, atol=1e-15)
    diag = [6, 12, 17, 21, 24, 26]
    assert np.allclose(rec_last[diag], own[diag], rtol=1e-9)
    scale = np.sqrt(np.outer(own[diag], own[diag]))[np.triu_indices(6)]
    assert np.all(np.abs(rec_last[6:] - own[6:]) <= 1e-9 * scale)


@pytest.mark.parametrize("prec", ["bf16", "f16", "fp32"])
def test_config3_full_size_sampled(hb, prec):
    """C3, N = 1e7, the bench's headline launch (and BJ's second run of C3 on the FFMA path, in the 8x8-register-tile
    shape the bench times): sampled particles vs the oracle, record vs the output."""
    desc, x = wl.config3(prec=prec)
    n = x.shape[1]
    assert n == 10_000_000
    out, rec = gpu_push_full(hb, desc, x)
    idx = sample_indices(n)
    ref, _ = oracle.push(desc, np.ascontiguousarray(x[:, idx]))
    assert np.all(np.isfinite(out))
    std = ref.std(axis=1)                      # G14: std of the oracle's output coordinate (over the sample)
    err = np.max(np.abs(out[:, idx].astype(np.float64) - ref), axis=1) / std
    print("C3 full size", prec, "max err/std on", idx.size, "sampled particles:", err)
    assert err.max() <= TOL[prec]
    check_moments(rec[-1], out)


def test_config2_full_size_sampled(hb):
    """conventional run at the size the HBM roofline is quoted on (N = 1e7, 500 elements in one fused pass)"""
    desc, x = wl.config2(n=10_000_000)
    out, rec = gpu_push_full(hb, desc, x)
    idx = sample_indices(x.shape[1])
    ref, _ = oracle.push(desc, np.ascontiguousarray(x[:, idx]))
    std = ref.std(axis=1)
    err = np.max(np.abs(out[:, idx].astype(np.float64) - ref), axis=1) / std
    print("C2 lattice N=1e7 max err/std:", err)
    assert err.max() <= 1e-6
    check_moments(rec[-1], out)


def test_config4_full_size_sampled(hb):
    """C4, N = 1e7, f16 operands, whole hybrid lattice (2 COORD_T stages + transport + chicane), free running"""
    desc, x = wl.config4(prec="f16")
    out, rec = gpu_push_full(hb, desc, x)
    idx = sample_indices(x.shape[1])
    ref, _ = oracle.push(desc, np.ascontiguousarray(x[:, idx]))
    assert np.all(np.isfinite(out))
    std = ref.std(axis=1)
    err = np.max(np.abs(out[:, idx].astype(np.float64) - ref), axis=1) / std
    print("C4 full size f16 free-running max err/std:", err)
    # two 16-bit stages in a row compound: reported, and held to the measured level (the per-stage contract, 2e-2 with
    # every stage fed from the oracle, is test_config4_full_size_every_stage_oracle_fed below)
    assert err.max() <= 5e-2
    assert rec.shape[0] == 4
    check_moments(rec[-1], out)


def test_config5_full_size_first_stage_and_run(hb):
    """C5's bunch (N = 1e8, 2.4 GB) through its first surrogate stage (6-512^4-6 tanh, streamed weights) and
    first transport section, f16 operands: sampled particles vs the oracle; then the whole 17-segment lattice in
    bf16 for finiteness and the record property."""
    desc, x = wl.config5(prec="f16")
    n = x.shape[1]
    assert n == 100_000_000
    first = wl.lattice(desc["elements"][:53])      # surrogate, monitor, 50 elements, monitor
    assert first["elements"][0]["kind"] == "surrogate" and first["elements"][-1]["kind"] == "monitor"
    out, rec = gpu_push_full(hb, first, x)
    idx = sample_indices(n)
    ref, _ = oracle.push(first, np.ascontiguousarray(x[:, idx]))
    std = ref.std(axis=1)
    err = np.max(np.abs(out[:, idx].astype(np.float64) - ref), axis=1) / std
    print("C5 N=1e8 stage 1 + run, f16, max err/std:", err)
    assert err.max() <= TOL["f16"]
    assert rec.shape[0] == 2
    del out
    desc_b, _ = wl.config5(prec="bf16", particles=False)
    out, rec = gpu_push_full(hb, desc_b, x)
    assert rec.shape[0] == 17 and np.all(np.isfinite(rec))
    sub = out[:, ::50]
    assert np.all(np.isfinite(sub))
    own = oracle.moments(np.ascontiguousarray(out[:, :5_000_000].astype(np.float64)))
    assert np.all(np.isfinite(own))
    # record of the whole bunch vs plain moments of a 5e6-particle prefix: statistical agreement only
    assert np.allclose(np.sqrt(rec[-1][[6, 17, 24]]), np.sqrt(own[[6, 17, 24]]), rtol=5e-2)


@pytest.mark.parametrize("name,width,hidden", [("P900", 900, 5), ("P700", 700, 3)])
def test_paper_shaped_nets_full_size_sampled(hb, name, width, hidden):
    """NEXT-1 at the paper's N (1e7) in the launch configuration `bench.py --workload P900|P700` times: the
    layered kernel (10 chunks x (hidden + 1) launches), f16 operands, sampled particles vs the oracle; record vs
    output; and the same bunch through hb_push_host (chunked host pipeline around the chunked layered stage)"""
    import torch
    desc, x = wl.paper_net(width, hidden, prec="f16")
    n = x.shape[1]
    assert n == 10_000_000 and hb.hb_surrogate_kernel("f16", desc["elements"][0]["widths"]) == "tcgen05-layered"
    out, rec = gpu_push_full(hb, desc, x)
    idx = sample_indices(n, m=3000)
    idx = np.unique(np.concatenate([idx, np.arange((1 << 20) - 300, (1 << 20) + 300)]))     # a chunk boundary
    ref, _ = oracle.push(desc, np.ascontiguousarray(x[:, idx]))
    assert np.all(np.isfinite(out))
    std = ref.std(axis=1)
    err = np.max(np.abs(out[:, idx].astype(np.float64) - ref), axis=1) / std
    print(name, "full size f16 max err/std on", idx.size, "sampled particles:", err)
    assert err.max() <= TOL["f16"]
    check_moments(rec[-1], out)
    lat = hb.Lattice.from_description(desc, device=0)
    host = torch.from_numpy(x.copy()).pin_memory()
    rec_h = lat.push_host(host, chunks=8)
    lat.close()
    assert np.array_equal(host.numpy(), out)
    assert np.allclose(rec_h[-1][:6], rec[-1][:6], rtol=1e-12, atol=1e-18)


# ------------------------------------------------------------------ every stage fed from the oracle, at full size
def full_size_oracle_fed(hb, desc, x, idx, renorm=False):
    """The whole bunch stays on the device and goes through the lattice piece by piece (tests/test_gpu_stagefed.py
    stage_lattices: every surrogate stage on its own, with the reference energy it has in the lattice).  The oracle
    carries the sampled particles `idx` in fp64; before every surrogate stage its state, rounded to fp32, is written
    over those particles of the device bunch, so the stage is oracle-fed on the sample while it runs in the launch
    configuration of the full size.  Returns per-stage max |gpu - oracle| / std(oracle output) over the sample."""
    import torch
    from test_gpu_stagefed import renormalised, stage_lattices
    c = hb.to_device(x)
    tidx = torch.from_numpy(idx).cuda()
    state = np.ascontiguousarray(x[:, idx].astype(np.float64))
    errs = []
    for sub, is_sur in stage_lattices(desc):
        fed = state.astype(np.float32)
        if is_sur and renorm:
            sub = renormalised(sub, fed)
        lat = hb.Lattice.from_description(sub, device=0)
        if is_sur:
            tf = torch.from_numpy(fed).cuda()
            for j in range(6):
                c[j].index_copy_(0, tidx, tf[j])
            ref, _ = oracle.push(sub, fed)
            lat.push(c)
            got = torch.stack([c[j].index_select(0, tidx) for j in range(6)]).cpu().numpy().astype(np.float64)
            assert np.all(np.isfinite(got))
            errs.append(np.max(np.abs(got - ref), axis=1) / ref.std(axis=1))
        else:
            lat.push(c)
        torch.cuda.synchronize()
        lat.close()
        state, _ = oracle.push(sub, state)
    del c
    torch.cuda.empty_cache()
    return np.array(errs)


def test_config4_full_size_every_stage_oracle_fed(hb):
    """C4, N = 1e7, f16: both COORD_T stages at 2e-2 (stage 2: 8 GeV incoming reference)"""
    desc, x = wl.config4(prec="f16")
    e = full_size_oracle_fed(hb, desc, x, sample_indices(x.shape[1]))
    print("C4 N=1e7 oracle-fed per-stage max err/std (f16):", e.max(axis=1))
    assert e.shape[0] == 2 and e.max() <= TOL["f16"]


def test_config5_full_size_every_stage_oracle_fed(hb):
    """C5 as specified (N = 1e8, 9 stages 6-512^4-6 tanh + 8 transport sections), f16: every stage at 2e-2, each
    normalised to the state the oracle feeds it (why: tests/test_gpu_stagefed.py::test_config5_every_stage_oracle_fed)"""
    desc, x = wl.config5(prec="f16")
    assert x.shape[1] == 100_000_000
    e = full_size_oracle_fed(hb, desc, x, sample_indices(x.shape[1], m=4000), renorm=True)
    print("C5 N=1e8 oracle-fed per-stage max err/std (f16):", e.max(axis=1))
    assert e.shape[0] == 9 and e.max() <= TOL["f16"]
