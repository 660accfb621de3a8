#!/usr/bin/env python
"""bench.py -- throughput of the hybrid-beamline hot path on B200 (one process per GPU).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C3|C4|C2|C5|P900|P700] [--impl hb|reference]

A step = one hb_push_moments of the whole lattice of the workload over one resident bunch.  Default
workload = BASELINE.json config 3 ("surrogate particles/s at 1e7; % of tensor peak": N = 1e7,
6-256^3-6 ReLU, 16-bit tensor cores, moments after the stage).  Default operand type is f16: the same
tcgen05.mma.kind::f16 instruction and rate as bf16, and the one that meets BASELINE.json's parity bound
(max |gpu - oracle| <= 2e-2 std; plain bf16 operands measure 4e-2..1.1e-1 on this net, see "parity" in
the line and DESIGN.md 6.5); `--prec bf16` times the bf16 variant, which the default run also reports
under "kernels".  The conventional-run kernel of the same metric ("particle-element pushes/s; % of HBM
peak") is measured in the same run at N = 1e7 and reported under "kernels" with its own roofline, as are
the bf16 / tf32 / fp32 variants and the C4 hybrid lattice.
Inputs (240 MB) exceed L2 (126 MB) and L2 is flushed between timed steps; the bunch is restored from a
pristine device copy before every step (outside the timed region) because the push is in place.
Timing: CUDA events on the launching stream, per step, summed; max over ranks.  One JSON line on stdout.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads as wl  # noqa: E402

METRIC = "particle-element pushes/s & surrogate particles/s at 1e7; % of HBM/tensor peak"
L2_FLUSH_BYTES = 256 << 20
TRAFFIC_FILE = os.path.join(ROOT, "profiles", "ncu_traffic.json")


def ncu_traffic(kernel, n):
    """dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of `kernel` at n particles, from the `ncu --set full`
    captures under profiles/ (profiles/ncu_traffic.json lists them: kernel, n, bytes, capture file, command); None if
    there is no capture of that kernel at that size"""
    try:
        for e in json.load(open(TRAFFIC_FILE))["entries"]:
            if e["kernel"] == kernel and int(e["n"]) == int(n):
                return float(e["dram_bytes"])
    except Exception:
        pass
    return None


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm_gbs": d["hbm_gbs"], "bf16_tflops": d["bf16_tflops"],
                "bf16_tflops_sustained": d.get("bf16_tflops_sustained", d["bf16_tflops"]), "source": "measured"}
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "source": "fallback"}


class ClockSampler:
    """nvidia-smi clocks line of B200_PROFILING.md, sampled every 5 ms during the timed region."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "5"], stdout=self.f,
                                      stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def count(self):
        try:
            self.f.flush()
            return sum(1 for _ in open(self.f.name))
        except Exception:
            return 0

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            c = [x.strip() for x in line.split(",")]
            if len(c) < 9:
                continue
            try:
                sm.append(float(c[1])); mx.append(float(c[2]))
            except ValueError:
                continue
            for nme, v in zip(names, c[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(nme)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), reasons=sorted(reasons), samples=len(sm))
        return out


def build_workload(name, prec, n):
    if name == "C3":
        desc, x = wl.config3(prec=prec, n=n or 10_000_000)
        label = "C3 surrogate-only: N=%d correlated Gaussian, MLP 6-256-256-256-6 ReLU He, %s, monitor after stage"
    elif name == "C4":
        desc, x = wl.config4(prec=prec, n=n or 10_000_000)
        label = "C4 hybrid: N=%d, 2 x [surrogate 6-128^3-6 tanh COORD_T %s + 9-element transport + 4-sbend chicane], 4 monitors"
    elif name == "C2":
        desc, x = wl.config2(n=n or 10_000_000)
        label = "C2 conventional-only: N=%d, 100 FODO cells (one fused run of 500 elements)%s, 1 monitor"
        prec = ""
    elif name == "C5":
        desc, x = wl.config5(prec=prec, n=n or 100_000_000)
        label = "C5 large bunch: N=%d, 9 x surrogate 6-512^4-6 tanh %s + 8 x 10 FODO cells, 17 monitors"
    elif name in ("P900", "P700"):
        w, h = (900, 5) if name == "P900" else (700, 3)
        desc, x = wl.paper_net(w, h, prec=prec, n=n or 10_000_000)
        label = "%s the paper's own network shape (P:177): N=%%d, one stage 6-%d^%d-6 PReLU %%s, random He weights, monitor after stage" % (name, w, h)
    else:
        raise SystemExit("unknown workload " + name)
    return desc, x, label % (x.shape[1], prec)


def count_work(desc):
    n_sur = sum(1 for e in desc["elements"] if e["kind"] == "surrogate")
    n_el = sum(1 for e in desc["elements"] if e["kind"] in ("drift", "quad", "sbend", "plens", "drift_exact", "quad_chromatic", "multipole"))
    flops = sum(wl.flops_per_particle(e["widths"]) for e in desc["elements"] if e["kind"] == "surrogate")
    return n_sur, n_el, flops


def segment_kinds(desc):
    """segment list as the library splits it: 'run' | 'sur' | 'mon' (standalone monitor)"""
    kinds, prev = [], None
    for e in desc["elements"]:
        k = e["kind"]
        if k == "monitor":
            if prev in ("run", "sur"):
                prev = "fusedmon"
            else:
                kinds.append("mon"); prev = "mon"
        elif k == "surrogate":
            kinds.append("sur"); prev = "sur"
        else:
            if prev != "run":
                kinds.append("run")
            prev = "run"
    return kinds


def timed_steps(torch, hb, lat, pristine, work, steps, warmup, flush, with_moments=True, segtimes=False):
    """returns (total_ms over `steps`, per-segment mean ms or None)"""
    rec = torch.empty((max(lat.num_monitors, 1), 27), dtype=torch.float64, device=work.device)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    seg_acc = None
    if segtimes:
        lat.enable_timing(True)
    for it in range(warmup + steps):
        work.copy_(pristine)
        flush.fill_(it & 0xff)                   # L2 flush: write a buffer larger than L2
        k = it - warmup
        if k >= 0:
            ev[k][0].record()
        if with_moments:
            lat.push_moments(work, out=rec)
        else:
            lat.push(work)
        if k >= 0:
            ev[k][1].record()
            if segtimes:
                t = np.array(lat.segment_times_ms())
                seg_acc = t if seg_acc is None else seg_acc + t
    torch.cuda.synchronize()
    if segtimes:
        lat.enable_timing(False)
    total = sum(a.elapsed_time(b) for a, b in ev)
    return total, (None if seg_acc is None else seg_acc / steps), rec


def oracle_rate(desc, x, budget_s, unit_count, gpu_head=None):
    """oracle (as it stands) on a bounded sample; returns (units/s, cores, sample description, parity).  parity: the
    oracle's output of that sample against the same particles of the timed GPU step (max |gpu - oracle| / std)"""
    import oracle
    n = x.shape[1]
    probe = min(n, 4096)
    t0 = time.perf_counter()
    oracle.push(desc, x[:, :probe])
    dt = max(time.perf_counter() - t0, 1e-4)
    ns = int(min(n, max(probe, (probe / dt) * budget_s)))
    ns = min(ns, 1 << 22)
    t0 = time.perf_counter()
    ref, _ = oracle.push(desc, x[:, :ns])
    dt = time.perf_counter() - t0
    parity = None
    if gpu_head is not None:
        m = min(ns, gpu_head.shape[1])
        ref = np.asarray(ref)[:, :m]
        err = np.max(np.abs(gpu_head[:, :m].astype(np.float64) - ref), axis=1) / ref.std(axis=1)
        parity = {"max_abs_err_over_std": [float(v) for v in err], "particles": int(m),
                  "against": "fp64 oracle, output of the last timed step"}
    return unit_count * ns / dt, oracle.num_threads(), "first %d particles of the workload, whole lattice, %.1f s" % (ns, dt), parity


def run_reference(args, rank, world):
    """--impl reference: the fp64 oracle on the host cores (rank 0 only)."""
    if rank != 0:
        return
    import oracle
    desc, x, label = build_workload(args.workload, args.prec, args.n)
    n_sur, n_el, flops = count_work(desc)
    units = n_sur if n_sur else n_el
    probe = min(x.shape[1], 2048)
    t0 = time.perf_counter()
    oracle.push(desc, x[:, :probe])
    rate = probe / max(time.perf_counter() - t0, 1e-4)
    per_step_s = max(0.5, min(10.0, 100.0 / (args.steps + args.warmup)))
    ns = int(max(256, min(x.shape[1], rate * per_step_s, 1 << 19)))
    xs = np.ascontiguousarray(x[:, :ns])
    for _ in range(args.warmup):
        oracle.push(desc, xs)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.push(desc, xs)
    dt = time.perf_counter() - t0
    value = units * ns * args.steps / dt
    unit = "surrogate particle-inferences/s" if n_sur else "particle-element pushes/s"
    sample = "each step = first %d particles of the workload through the whole lattice" % ns
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": unit, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic (seeded; see DESIGN.md)",
        "config": {"workload": label, "sample": sample},
        "cpu_baseline": {"value": value, "unit": unit, "cores": oracle.num_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": unit, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def kernel_extras(torch, hb, args, pk, flush, dev, dp):
    """per-kernel measurements at N = 1e7 beside the headline step.  dp: hb_device_peaks() of this device (measured pipe
    rates: the ALU-bound kernels and the tf32 mode are quoted against them)"""
    tf32_peak = pk["bf16_tflops"] * dp["mma_tf32_tflops"] / dp["mma_f16_tflops"]
    tf32_src = pk["source"] + " bf16 x %.3f (kind::tf32 : kind::f16 rate of the tensor pipe measured by hb_device_peaks: %.0f / %.0f TFLOP/s)" % (
        dp["mma_tf32_tflops"] / dp["mma_f16_tflops"], dp["mma_tf32_tflops"], dp["mma_f16_tflops"])
    p16 = args.prec if args.prec in ("f16", "bf16") else "f16"      # 16-bit operand type of the tensor-core extras
    out = []
    n = args.n or 10_000_000
    reps = 10

    PARITY_N = 100_000

    def measure(desc, xh, label, with_moments, steps=reps, run_mode="composed", prec=None, parity=False):
        """mean ms per step, per-segment ms [, max |gpu - oracle| / std(oracle) per coordinate over the first PARITY_N
        particles of the last timed step]"""
        lat = hb.Lattice.from_description(desc, run_mode=run_mode, device=dev.index, prec=prec)
        pristine = torch.from_numpy(xh).to(dev)
        work = torch.empty_like(pristine)
        tot, seg, _ = timed_steps(torch, hb, lat, pristine, work, steps, 3, flush, with_moments=with_moments, segtimes=True)
        lat.close()
        par = None
        if parity:
            import oracle
            m = min(PARITY_N, xh.shape[1])
            d2 = dict(desc)
            if prec is not None:      # the oracle ignores the precision; keep the description as it is
                pass
            ref, _ = oracle.push(d2, np.ascontiguousarray(xh[:, :m]))
            got = work[:, :m].cpu().numpy().astype(np.float64)
            err = np.max(np.abs(got - ref), axis=1) / ref.std(axis=1)
            par = {"max_abs_err_over_std": float(err.max()), "particles": int(m)}
        del pristine, work
        return (tot / steps, seg, par) if parity else (tot / steps, seg)

    # (a) conventional run kernel, C2 lattice (500 elements) at N = 1e7: composed (HBM-bound)
    desc2, x2 = wl.config2(n=n)
    for mom in (False, True):
        ms, seg = measure(desc2, x2, "run", mom)
        k_ms = float(seg[0])
        gbs = 48.0 * n / (k_ms * 1e-3) / 1e9
        out.append({"kernel": "hb_run_composed_kernel" + ("<moments>" if mom else ""), "workload": "C2 lattice (500 elements, one run), N=%d" % n,
                    "ms": k_ms, "particle_element_pushes_per_s": 500.0 * n / (k_ms * 1e-3),
                    "roofline": {"bound": "hbm", "achieved": gbs, "peak": pk["hbm_gbs"], "unit": "GB/s",
                                 "frac": gbs / pk["hbm_gbs"], "traffic": ncu_traffic("hb_run_composed_kernel", n),
                                 "peak_source": pk["source"]}})
    # same kernel at N = 1e8 (2.4 GB per bunch, 4.8 GB of traffic per launch): launch + event overhead (~6 us) no
    # longer visible beside 730 us of streaming
    if not args.n:
        nb = 100_000_000
        xb = wl.gaussian_bunch(nb, 2)
        for mom in (False, True):
            lat = hb.Lattice.from_description(desc2, run_mode="composed", device=dev.index)
            pristine = torch.from_numpy(xb).to(dev)
            work = torch.empty_like(pristine)
            tot, seg, _ = timed_steps(torch, hb, lat, pristine, work, 5, 3, flush, with_moments=mom, segtimes=True)
            lat.close()
            del pristine, work
            k_ms = float(seg[0])
            gbs = 48.0 * nb / (k_ms * 1e-3) / 1e9
            out.append({"kernel": "hb_run_composed_kernel" + ("<moments>" if mom else ""),
                        "workload": "C2 lattice (500 elements, one run), N=%d" % nb, "ms": k_ms,
                        "particle_element_pushes_per_s": 500.0 * nb / (k_ms * 1e-3),
                        "roofline": {"bound": "hbm", "achieved": gbs, "peak": pk["hbm_gbs"], "unit": "GB/s",
                                     "frac": gbs / pk["hbm_gbs"], "traffic": None, "peak_source": pk["source"]}})
        del xb
    # sequential (fp64 registers, ALU-bound): 2700 DFMA-class ops per particle
    ms, seg = measure(desc2, x2, "run", False, steps=5, run_mode="sequential")
    k_ms = float(seg[0])
    dp_peak = dp["dfma_tfma"]             # measured fp64 FMA rate of this device (hb_device_peaks)
    ach = 2700.0 * n / (k_ms * 1e-3) / 1e12
    out.append({"kernel": "hb_run_sequential_kernel<double>", "workload": "C2 lattice, N=%d" % n, "ms": k_ms,
                "particle_element_pushes_per_s": 500.0 * n / (k_ms * 1e-3),
                "roofline": {"bound": "alu", "achieved": ach, "peak": dp_peak, "unit": "TFMA/s (fp64)", "frac": ach / dp_peak,
                             "traffic": None, "peak_source": "measured: hb_device_peaks fp64 FMA chains"}})
    # non-linear run (NEXT-3): 100 chromatic FODO cells = 300 exact drifts + 200 chromatic quadrupoles, always on the
    # fp64 sequential kernel (sin/cos/sqrt per particle and element: ALU/MUFU-bound, no closed-form FMA count)
    cell = [wl.drift_exact(0.25), wl.quad_chromatic(0.1, 1.2), wl.drift_exact(0.5), wl.quad_chromatic(0.1, -1.2), wl.drift_exact(0.25)]
    descn = wl.lattice(cell * 100 + [wl.monitor()])
    ms, seg = measure(descn, x2, "run", True, steps=3)
    k_ms = float(seg[0])
    out.append({"kernel": "hb_run_sequential_kernel<double> (non-linear elements)", "workload": "100 chromatic FODO cells, N=%d" % n,
                "ms": k_ms, "particle_element_pushes_per_s": 500.0 * n / (k_ms * 1e-3)})
    del x2
    # (b) surrogate C3 with the other 16-bit operand type (same instruction, same rate), tf32 and fp32 FFMA
    if args.workload == "C3":
        other = "bf16" if args.prec == "f16" else "f16"
        desc3, x3 = wl.config3(prec=other, n=n)
        fl = wl.flops_per_particle(desc3["elements"][0]["widths"])
        ms, seg, par = measure(desc3, x3, "sur", True, parity=True)
        k_ms = float(seg[0])
        tf = fl * n / (k_ms * 1e-3) / 1e12
        out.append({"kernel": "hb_sur_tc2_kernel<%s>" % other, "workload": "C3, N=%d" % n, "ms": k_ms,
                    "particle_inferences_per_s": n / (k_ms * 1e-3), "parity": par,
                    "parity_bound": "2e-2 (BASELINE.json); plain bf16 operands are outside it: reported, not conforming (DESIGN.md 6.5)",
                    "roofline": {"bound": "tensor", "achieved": tf, "peak": pk["bf16_tflops"], "unit": "TFLOP/s",
                                 "frac": tf / pk["bf16_tflops"], "traffic": ncu_traffic("hb_sur_tc2_kernel", n),
                                 "peak_source": pk["source"]}})
        ms, seg, par = measure(desc3, x3, "sur", True, steps=5, prec="tf32", parity=True)
        k_ms = float(seg[0])
        tf = fl * n / (k_ms * 1e-3) / 1e12
        out.append({"kernel": "hb_sur_tcs_kernel<tf32>", "workload": "C3, N=%d" % n, "ms": k_ms,
                    "particle_inferences_per_s": n / (k_ms * 1e-3), "parity": par, "parity_bound": "2e-2",
                    "roofline": {"bound": "tensor", "achieved": tf, "peak": tf32_peak, "unit": "TFLOP/s",
                                 "frac": tf / tf32_peak, "traffic": None, "peak_source": tf32_src}})
        ms, seg, par = measure(desc3, x3, "sur", True, steps=2, prec="fp32", parity=True)
        k_ms = float(seg[0])
        fma_peak = dp["ffma_tfma"]
        ach = 0.5 * fl * n / (k_ms * 1e-3) / 1e12
        out.append({"kernel": "hb_sur_fp32_kernel", "workload": "C3, N=%d" % n, "ms": k_ms,
                    "particle_inferences_per_s": n / (k_ms * 1e-3), "parity": par, "parity_bound": "1e-5",
                    "roofline": {"bound": "alu", "achieved": ach, "peak": fma_peak, "unit": "TFMA/s (fp32)",
                                 "frac": ach / fma_peak, "traffic": None,
                                 "peak_source": "measured: hb_device_peaks fp32 FMA chains"}})
        del x3
        # (b2) one C5 stage (6-512^4-6 tanh, weights streamed from L2) at N = 1e7
        desc5, _ = wl.config5(prec=p16, particles=False)
        d5 = wl.lattice(desc5["elements"][:2])
        x5 = wl.gaussian_bunch(n, 5)
        fl5 = wl.flops_per_particle(d5["elements"][0]["widths"])
        ms, seg = measure(d5, x5, "sur", True, steps=5)
        k_ms = float(seg[0])
        tf = fl5 * n / (k_ms * 1e-3) / 1e12
        out.append({"kernel": "hb_sur_tcs_kernel<%s> (streamed weights)" % p16, "workload": "one C5 stage 6-512^4-6 tanh, N=%d" % n, "ms": k_ms,
                    "particle_inferences_per_s": n / (k_ms * 1e-3),
                    "roofline": {"bound": "tensor", "achieved": tf, "peak": pk["bf16_tflops"], "unit": "TFLOP/s",
                                 "frac": tf / pk["bf16_tflops"], "frac_of_sustained": tf / pk["bf16_tflops_sustained"],
                                 "traffic": ncu_traffic("hb_sur_tcs_kernel", n), "peak_source": pk["source"]}})
        del x5
        # (b3) the paper's own network shapes on the layered kernel, one stage at N = 1e7; the paper's timings
        # (P:199, 1 x A100, PyTorch) are context, not the target
        for wname, (wd, hd, paper_ms) in (("P900", (900, 5, 1120.0)), ("P700", (700, 3, 494.0))):
            descp, xp = wl.paper_net(wd, hd, prec=p16, n=n)
            flp = wl.flops_per_particle(descp["elements"][0]["widths"])
            ms, seg = measure(descp, xp, "sur", True, steps=3)
            k_ms = float(seg[0])
            tf = flp * n / (k_ms * 1e-3) / 1e12
            out.append({"kernel": "hb_sur_tcw_kernel<%s> (%d launches: one per layer and 2^20-particle chunk)" % (p16, (hd + 1) * ((n + (1 << 20) - 1) >> 20)),
                        "workload": "%s: one stage 6-%d^%d-6 PReLU, N=%d" % (wname, wd, hd, n), "ms": k_ms,
                        "particle_inferences_per_s": n / (k_ms * 1e-3), "paper_ms_per_stage_a100": paper_ms if n == 10_000_000 else None,
                        "roofline": {"bound": "tensor", "achieved": tf, "peak": pk["bf16_tflops"], "unit": "TFLOP/s",
                                     "frac": tf / pk["bf16_tflops"], "frac_of_sustained": tf / pk["bf16_tflops_sustained"],
                                     "traffic": None, "peak_source": pk["source"]}})
            del xp
        # (c) C4 hybrid lattice (all rows a1-a7 in one push)
        desc4, x4 = wl.config4(prec=p16, n=n)
        ms, seg = measure(desc4, x4, "c4", True)
        fl4 = wl.flops_per_particle([6, 128, 128, 128, 6])
        kinds = segment_kinds(desc4)
        sur_ms = float(np.mean([t for t, k in zip(seg, kinds) if k == "sur"]))
        run_ms = float(np.mean([t for t, k in zip(seg, kinds) if k == "run"]))
        # a 6-128^3-6 tanh stage is bound by the special-function unit (16 tanh/clk/SM), not by the tensor pipe:
        # 384 tanh per particle
        xu_peak = dp["tanh_tps"]
        xu_ach = 384.0 * n / (sur_ms * 1e-3) / 1e12
        out.append({"kernel": "C4 whole push (2 surrogate + 2 run kernels + 4 moment finalizes)", "workload": "C4, N=%d" % n,
                    "ms": ms, "particles_per_s": n / (ms * 1e-3), "surrogate_ms": sur_ms, "run_ms": run_ms,
                    "surrogate_tflops": fl4 * n / (sur_ms * 1e-3) / 1e12, "run_gbs": 48.0 * n / (run_ms * 1e-3) / 1e9,
                    "roofline": {"bound": "alu", "achieved": xu_ach, "peak": xu_peak, "unit": "Ttanh/s (MUFU, surrogate kernel)",
                                 "frac": xu_ach / xu_peak, "traffic": ncu_traffic("hb_sur_tc_kernel", n),
                                 "peak_source": "measured: hb_device_peaks tanh.approx chains"}})
        del x4
        # (d) NEXT-4: K candidate settings of one transport gap over the same resident bunch (hb_push_candidates): one
        # pass over the particles whatever K is
        gap = wl.lattice([wl.drift(0.5), wl.plens(0.05, 10.0), wl.drift(0.45), wl.monitor()], kinetic_MeV=8000.0)
        latg = hb.Lattice.from_description(gap, device=dev.index)
        xg = torch.from_numpy(wl.gaussian_bunch(n, 6)).to(dev)
        K = 256
        rng = np.random.default_rng(1)
        d0 = rng.uniform(0.05, 0.9, K)
        length = np.stack([d0, np.full(K, 0.05), 0.95 - d0], axis=1)
        param = np.stack([np.zeros(K), rng.uniform(0.0, 40.0, K), np.zeros(K)], axis=1)
        recs = torch.empty((K, 27), dtype=torch.float64, device=dev)
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(reps)]
        for it in range(3 + reps):
            flush.fill_(it & 0xff)
            if it >= 3:
                evs[it - 3][0].record()
            latg.push_candidates(xg, [0, 1, 2], length, param, out=recs)
            if it >= 3:
                evs[it - 3][1].record()
        torch.cuda.synchronize()
        c_ms = sum(a.elapsed_time(b) for a, b in evs) / reps
        latg.close()
        del xg
        gbs = 24.0 * n / (c_ms * 1e-3) / 1e9
        out.append({"kernel": "hb_push_candidates (moment partials + finalize + hb_candidates_kernel)",
                    "workload": "%d candidate settings of a drift / plasma lens / drift gap, N=%d, bunch read once" % (K, n),
                    "ms": c_ms, "candidate_evaluations_per_s": K / (c_ms * 1e-3),
                    "roofline": {"bound": "hbm", "achieved": gbs, "peak": pk["hbm_gbs"], "unit": "GB/s (read only: 24 B per particle)",
                                 "frac": gbs / pk["hbm_gbs"], "traffic": None, "peak_source": pk["source"] + " (copy bandwidth)"}})
        # (d2) launch-bound case: C1 (N = 4096: FODO cell | 6-64-64-6 tanh stage | drift, three monitors = 6 launches of a
        # few microseconds each).  A push only enqueues (no allocation, no host synchronisation), so it can be captured
        # into a CUDA graph once and replayed: pushes back to back on one stream, direct launches against graph replays.
        desc1, x1 = wl.config1(prec=p16)
        lat1 = hb.Lattice.from_description(desc1, device=dev.index)
        w1 = torch.from_numpy(x1).to(dev)
        rec1 = torch.zeros((lat1.num_monitors, 27), dtype=torch.float64, device=dev)
        nrep = 200
        for _ in range(20):
            lat1.push_moments(w1, out=rec1)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(nrep):
            lat1.push_moments(w1, out=rec1)
        e1.record()
        torch.cuda.synchronize()
        direct_us = e0.elapsed_time(e1) * 1e3 / nrep
        graph = torch.cuda.CUDAGraph()
        side = torch.cuda.Stream(device=dev)
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):
            with torch.cuda.graph(graph, stream=side):
                lat1.push_moments(w1, out=rec1)
        torch.cuda.synchronize()
        for _ in range(20):
            graph.replay()
        torch.cuda.synchronize()
        e0.record()
        for _ in range(nrep):
            graph.replay()
        e1.record()
        torch.cuda.synchronize()
        graph_us = e0.elapsed_time(e1) * 1e3 / nrep
        nl1 = lat1.num_launches(True, x1.shape[1])
        lat1.close()
        out.append({"kernel": "C1 whole push, launch-bound (%d launches): direct launches vs one CUDA-graph replay" % nl1,
                    "workload": "C1: N=%d, FODO cell | 6-64-64-6 tanh %s | drift, 3 monitors; %d pushes back to back" % (x1.shape[1], p16, nrep),
                    "ms": graph_us * 1e-3, "us_per_push_direct": direct_us, "us_per_push_graph_replay": graph_us,
                    "particles_per_s": x1.shape[1] / (graph_us * 1e-6)})
        # (e) C5 as BASELINE.json specifies it: N = 1e8 (2.4 GB bunch), 9 streamed-weights stages + 8 runs + 17 monitors
        if not args.n:
            desc5f, x5f = wl.config5(prec=p16, n=100_000_000)
            ms, seg = measure(desc5f, x5f, "c5", True, steps=2)
            kinds5 = segment_kinds(desc5f)
            sur5 = float(np.mean([t for t, k in zip(seg, kinds5) if k == "sur"]))
            run5 = float(np.mean([t for t, k in zip(seg, kinds5) if k == "run"]))
            nb = x5f.shape[1]
            tf = fl5 * nb / (sur5 * 1e-3) / 1e12
            out.append({"kernel": "C5 whole push (9 x hb_sur_tcs_kernel + 8 x hb_run_composed_kernel + 17 finalizes)",
                        "workload": "C5 as specified: N=%d, 9 x 6-512^4-6 tanh %s + 8 x 10 FODO cells, 17 monitors" % (nb, p16),
                        "ms": ms, "particles_per_s": nb / (ms * 1e-3), "surrogate_inferences_per_s": 9.0 * nb / (ms * 1e-3),
                        "surrogate_ms": sur5, "run_ms": run5, "run_gbs": 48.0 * nb / (run5 * 1e-3) / 1e9,
                        "roofline": {"bound": "tensor", "achieved": tf, "peak": pk["bf16_tflops"], "unit": "TFLOP/s (one stage)",
                                     "frac": tf / pk["bf16_tflops"], "frac_of_sustained": tf / pk["bf16_tflops_sustained"],
                                     "traffic": None, "peak_source": pk["source"]}})
            del x5f
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="hb", choices=["hb", "reference"])
    ap.add_argument("--workload", default="C3")
    ap.add_argument("--prec", default="f16")
    ap.add_argument("--n", type=int, default=0, help="override particle count (testing)")
    ap.add_argument("--no-extras", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "hb" else args.warmup
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import torch
    import torch.distributed as dist
    import paper_2402_17248_b200 as hb
    hb.lib()                                   # fail loudly if the CUDA library is missing
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    pk = peaks()
    dp = hb.hb_device_peaks(local)             # measured pipe rates of this device (fp32 / fp64 FMA, tanh, tensor f16 / tf32)

    desc, x, label = build_workload(args.workload, args.prec, args.n)
    if world > 1:   # weak scaling: every rank pushes its own bunch of the full size (particles shard)
        x = np.roll(x, rank * 1009, axis=1)
    n = x.shape[1]
    n_sur, n_el, flops = count_work(desc)
    lat = hb.Lattice.from_description(desc, device=local)
    host = torch.from_numpy(x).pin_memory()
    pristine = host.to(dev)
    work = torch.empty_like(pristine)
    flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device=dev)

    # ---- timed region: K steps, device time, barrier + synchronize on both sides
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    sampler = ClockSampler(local)
    total_ms, seg_ms, rec = timed_steps(torch, hb, lat, pristine, work, args.steps, args.warmup, flush, True, True)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    in_region = sampler.count()
    # nvidia-smi answers a query in tens of milliseconds, a 20-step region lasts ~50: the same step goes on, untimed,
    # until the sampler has watched >= 0.5 s of it (clocks and throttle reasons under this very load)
    t_watch = time.perf_counter()
    while time.perf_counter() - t_watch < 0.5:
        timed_steps(torch, hb, lat, pristine, work, 5, 0, flush, True, False)
    clocks = sampler.stop()
    clocks["samples_in_timed_region"] = in_region
    clocks["note"] = "sampled over the timed region and 0.5 s more of the same step"
    t = torch.tensor([total_ms], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    total_ms = float(t.item())
    ms_step = total_ms / args.steps
    assert bool(torch.isfinite(rec).all()), "non-finite moments"
    merged_ok = None
    if world > 1:       # monitor records of the whole N-rank bunch: 224 B per monitor and rank, outside the timed region
        try:
            merged = hb.allgather_merge_records(rec, n)
            merged_ok = bool(np.isfinite(merged).all())
        except Exception as ex:                     # reported, never fatal to the timing line
            merged_ok = "failed: %s" % (ex,)

    # ---- end to end through the C ABI with HOST buffers: hb_push_host (pinned host arrays in, results and moment
    # records back in host memory when the call returns; H2D, kernels, D2H pipelined in chunks inside the library).
    # The call is synchronous, so it is timed with the host clock; the bunch is restored between steps (untimed).
    e2e_steps = max(2, min(args.steps, 5))
    e2e_chunks = 8
    host_work = torch.empty_like(host).pin_memory()
    e2e_total = 0.0
    for it in range(1 + e2e_steps):
        host_work.copy_(host)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        rec_host = lat.push_host(host_work, chunks=e2e_chunks)
        dt = time.perf_counter() - t0
        if it > 0:
            e2e_total += dt
    assert rec_host is None or bool(np.isfinite(rec_host).all()), "non-finite host records"
    e2e_ms = torch.tensor([1e3 * e2e_total / e2e_steps], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(e2e_ms, op=dist.ReduceOp.MAX)
    e2e_ms = float(e2e_ms.item())
    rec_bytes = 0 if rec_host is None else int(rec_host.size * 8)

    units = n_sur if n_sur else n_el
    unit = "surrogate particle-inferences/s" if n_sur else "particle-element pushes/s"
    value = units * n * world / (ms_step * 1e-3)
    e2e_value = units * n * world / (e2e_ms * 1e-3)

    # ---- roofline of the dominant kernel (live per-segment CUDA-event times of the timed steps)
    kinds = segment_kinds(desc)
    dom = int(np.argmax(seg_ms))
    dom_ms = float(seg_ms[dom])
    if kinds[dom] == "sur":
        per = flops / max(n_sur, 1)
        ach = per * n / (dom_ms * 1e-3) / 1e12
        widest = max(max(e["widths"][1:-1]) for e in desc["elements"] if e["kind"] == "surrogate")
        kname = "hb_sur_tcw_kernel" if widest > 512 else ("hb_sur_tcs_kernel" if widest > 256 else
                                                          ("hb_sur_tc2_kernel" if widest > 128 else "hb_sur_tc_kernel"))
        if args.prec == "fp32":
            # FFMA path on the CUDA cores: peak derived in DESIGN.md 6.3 (148 SMs x 128 lanes x 1.965 GHz)
            fma_peak = dp["ffma_tfma"]
            ach = 0.5 * per * n / (dom_ms * 1e-3) / 1e12
            roof = {"bound": "alu", "achieved": ach, "peak": fma_peak, "unit": "TFMA/s (fp32)", "frac": ach / fma_peak,
                    "traffic": None, "kernel": "hb_sur_fp32_kernel", "kernel_ms": dom_ms,
                    "peak_source": "measured: hb_device_peaks fp32 FMA chains",
                    "algorithmic_fma_per_particle": 0.5 * per}
        elif args.prec == "tf32":
            t32 = pk["bf16_tflops"] * dp["mma_tf32_tflops"] / dp["mma_f16_tflops"]
            roof = {"bound": "tensor", "achieved": ach, "peak": t32, "unit": "TFLOP/s",
                    "frac": ach / t32, "traffic": None, "kernel": "hb_sur_tcs_kernel",
                    "kernel_ms": dom_ms, "peak_source": pk["source"] + " bf16 x measured kind::tf32 : kind::f16 pipe ratio (hb_device_peaks)",
                    "algorithmic_flop_per_particle": per}
        else:
            roof = {"bound": "tensor", "achieved": ach, "peak": pk["bf16_tflops"], "unit": "TFLOP/s",
                    "frac": ach / pk["bf16_tflops"], "traffic": ncu_traffic(kname, n), "kernel": kname,
                    "kernel_ms": dom_ms, "peak_source": pk["source"] + " (burst, cuBLAS bf16; f16 and bf16 share tcgen05.mma.kind::f16 and its peak)",
                    "frac_of_sustained": ach / pk["bf16_tflops_sustained"],
                    "algorithmic_flop_per_particle": per}
    else:
        ach = 48.0 * n / (dom_ms * 1e-3) / 1e9
        roof = {"bound": "hbm", "achieved": ach, "peak": pk["hbm_gbs"], "unit": "GB/s", "frac": ach / pk["hbm_gbs"],
                "traffic": ncu_traffic("hb_run_composed_kernel", n), "kernel": "hb_run_composed_kernel",
                "kernel_ms": dom_ms, "peak_source": pk["source"]}

    # BASELINE.md holds the paper's number only for its own network shapes at N = 1e7 (P:199, 1 x A100: context)
    paper_rate = {"P900": 1e7 / 1.12, "P700": 1e7 / 0.494}.get(args.workload) if n == 10_000_000 and world == 1 else None
    line = {
        "metric": METRIC, "value": value, "unit": unit, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": (value / paper_rate) if paper_rate else None,
        "dtype": args.prec if n_sur else "f32", "data": "synthetic (seeded; shapes of the paper's workloads, DESIGN.md)",
        "config": {"workload": label, "l2": "inputs (%d MB) exceed L2 and a 256 MB buffer is written between timed steps" % (24 * n // 1000000),
                   "timing": "CUDA events per step on the launching stream, summed; max over ranks", "parallelism": "particles sharded, no collective"},
        "element_pushes_per_s": n_el * n * world / (ms_step * 1e-3),
        "particles_per_s": n * world / (ms_step * 1e-3),
        "segment_ms": [float(v) for v in seg_ms],
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": unit, "h2d_bytes_per_step": int(host.numel() * 4),
                "d2h_bytes_per_step": int(host.numel() * 4 + rec_bytes), "ms_per_step": e2e_ms,
                "api": "hb_push_host(chunks=%d): pinned host arrays, synchronous, host clock" % e2e_chunks},
        "gpu_launches": int(args.steps * lat.num_launches(True, n)),
        "records_merged_over_ranks": merged_ok,
        "roofline": roof,
        "device_peaks": dp,
    }
    gpu_head = work[:, :1 << 22].cpu().numpy() if (rank == 0 and world == 1 and not args.no_cpu_baseline) else None
    lat.close()
    del host_work
    if rank == 0 and world == 1:
        if not args.no_extras:
            del pristine, work
            line["kernels"] = kernel_extras(torch, hb, args, pk, flush, dev, dp)
        if not args.no_cpu_baseline:
            v, cores, sample, parity = oracle_rate(desc, x, 12.0, units, gpu_head)
            line["cpu_baseline"] = {"value": v, "unit": unit, "cores": cores, "kind": "oracle", "sample": sample}
            line["parity"] = parity
            line["paper_context"] = "paper: 632 ms/stage at N=1e7 on 1 x A100 (PAPER.md P:197), 1.58e7 particle-inferences/s; other nets, other hardware"
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(line))


if __name__ == "__main__":
    main()
