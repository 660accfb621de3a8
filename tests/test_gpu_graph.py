"""A push is enqueue-only (caller's stream, no host synchronisation, nothing allocated per push), so it
can be captured into a CUDA graph and replayed (-m gpu).  torch is used for the graph object, streams and memory only."""
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


def test_push_moments_captured_and_replayed(hb):
    """hybrid lattice (run, surrogate stage on the tensor cores, run, three monitors): the replayed graph gives the bits
    of the directly enqueued push, twice, and agrees with the oracle"""
    import torch
    desc, x = wl.config4(prec="f16", n=20_000, stages=1)
    ref, ref_rec = oracle.push(desc, x)
    lat = hb.Lattice.from_description(desc, device=0)
    pristine = torch.stack(hb.to_device(x))                      # [6, n] on the device
    work = hb.to_device(x)
    rec = torch.zeros((lat.num_monitors, 27), dtype=torch.float64, device="cuda:0")
    # direct push
    lat.push_moments(work, out=rec)
    torch.cuda.synchronize()
    direct = hb.to_host(work).copy()
    direct_rec = rec.cpu().numpy().copy()
    # capture one push on a side stream
    g = torch.cuda.CUDAGraph()
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        for j in range(6):
            work[j].copy_(pristine[j])
        lat.push_moments(work, out=rec)                            # warm-up on the capture stream
        torch.cuda.synchronize()
        with torch.cuda.graph(g, stream=s):
            lat.push_moments(work, out=rec)
    torch.cuda.synchronize()
    for _ in range(2):
        for j in range(6):
            work[j].copy_(pristine[j])
        rec.zero_()
        torch.cuda.synchronize()
        g.replay()
        torch.cuda.synchronize()
        assert np.array_equal(hb.to_host(work), direct)
        assert np.array_equal(rec.cpu().numpy(), direct_rec)
    got = direct.astype(np.float64)
    assert np.max(np.abs(got - ref) / ref.std(axis=1, keepdims=True)) <= 2e-2
    lat.close()


def test_cluster_kernel_and_static_moments_captured(hb):
    """the N-half kernel (CTA pairs, hb_sur_tc2.cu) and the no-allocation moments entry point inside one graph"""
    import torch
    desc, x = wl.config3(prec="f16", n=30_000)
    lat = hb.Lattice.from_description(desc, device=0)
    assert hb.hb_surrogate_kernel("f16", [6, 256, 256, 256, 6]) == "tcgen05-resident"
    pristine = torch.stack(hb.to_device(x))
    work = hb.to_device(x)
    rec = torch.zeros((lat.num_monitors, 27), dtype=torch.float64, device="cuda:0")
    rec_static = torch.zeros(27, dtype=torch.float64, device="cuda:0")
    lat.push_moments(work, out=rec)
    hb.moments_static(work, rec_static)                            # first call on the device: looks the scratch address up
    torch.cuda.synchronize()
    direct = hb.to_host(work).copy()
    direct_rec = rec.cpu().numpy().copy()
    direct_static = rec_static.cpu().numpy().copy()
    g = torch.cuda.CUDAGraph()
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        with torch.cuda.graph(g, stream=s):
            lat.push_moments(work, out=rec)
            hb.moments_static(work, rec_static)
    torch.cuda.synchronize()
    for j in range(6):
        work[j].copy_(pristine[j])
    rec.zero_()
    rec_static.zero_()
    torch.cuda.synchronize()
    g.replay()
    torch.cuda.synchronize()
    assert np.array_equal(hb.to_host(work), direct)
    assert np.array_equal(rec.cpu().numpy(), direct_rec)
    assert np.array_equal(rec_static.cpu().numpy(), direct_static)
    # the monitor behind the stage and the standalone pass see the same bunch
    assert np.allclose(direct_static, direct_rec[-1], rtol=1e-9, atol=1e-18)
    lat.close()
