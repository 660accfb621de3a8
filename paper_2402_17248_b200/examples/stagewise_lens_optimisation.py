#!/usr/bin/env python
"""Stage-by-stage optimisation of the transport gaps of a staged beamline.

The paper transports the beam from one plasma stage to the next through a gap with one (plasma) lens whose position and
strength are free: 2 (N_stage - 1) = 28 parameters for 15 stages, optimised "in a stage-by-stage sequence" with
Nelder-Mead, one tracking run per evaluation of the objective.  This example runs that sequence on a synthetic
15-stage line through the C ABI:

    stage j      a surrogate stage F_nn (random weights stand in for the trained ones, which are not available),
                 COORD_T, +7 GeV per stage
    gap j        drift d, plasma lens (length 5 cm, strength k), drift 1 m - d           <- the two free parameters

For gap j the bunch behind stage j is resident on the device and every Nelder-Mead step asks for the objective at a
batch of candidate (d, k): `Lattice.push_candidates` evaluates the whole batch in ONE pass over the bunch
(hb_push_candidates: the gap's elements concatenated per candidate on the host in fp64, the bunch read once, one
27-double record per candidate), so an evaluation costs three small launches whatever the bunch size is.  The
objective asks for a matched beam at the entrance of the next stage: size and divergence in both planes, each in units
of its nominal value (the divergence's shrinks with the reference momentum), summed -- the trained stages of the paper
would give the emittance behind the next stage instead; with random networks that has no meaning.  When a gap is
optimised its elements are set (hb_lattice_set_element), the bunch is pushed through it and through the next stage,
and the sequence moves on.

    python -m paper_2402_17248_b200.examples.stagewise_lens_optimisation [--stages 15] [--n 1000000]

Needs a B200 and scipy.  Prints the optimised parameters per gap and the evaluation rate.
"""
from __future__ import annotations

import argparse
import math
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads as wl  # noqa: E402


def stage_description(j, bg_in, bg_out, sd):
    """A stage that behaves like one: identity in the normalised fixed-time coordinates (PReLU net initialised to the
    identity, the construction of the oracle's identity pin) plus a small random non-linear perturbation, and the
    reference moved up by 7 GeV -- so transverse momenta are kept and the divergence shrinks (adiabatic damping)."""
    rng = np.random.default_rng([15, 1, j])
    H, eps = 128, 0.02
    A0 = np.zeros((H, 6)); A0[:6] = np.eye(6); A0 += eps * rng.standard_normal((H, 6))
    mid = []
    for _ in range(2):
        A = np.zeros((H, H)); A[:6, :6] = np.eye(6); A += eps / math.sqrt(H) * rng.standard_normal((H, H))
        mid.append(A)
    A3 = np.zeros((6, H)); A3[:, :6] = np.eye(6); A3 += eps / math.sqrt(H) * rng.standard_normal((6, H))
    W = [a.astype(np.float32) for a in [A0] + mid + [A3]]
    b = [(0.01 * rng.standard_normal(w.shape[0])).astype(np.float32) for w in W]
    mu_in = np.array([0, 0, 0, 0, 0, bg_in], dtype=np.float64)
    mu_out = np.array([0, 0, 0, 0, 0, bg_out], dtype=np.float64)
    return wl.surrogate([6, H, H, H, 6], W, b, "prelu", mu_in, sd, mu_out, sd, coord="t", prelu_a=[0.8, 0.8, 0.8],
                        ref_bg_out=bg_out, ref_z_out=0.0, prec="f16")


def gap_description(d, k):
    return [wl.drift(d), wl.plens(0.05, k), wl.drift(1.0 - d), wl.monitor()]


def nelder_mead_batched(f_batch, x0, step, iters=40):
    """Nelder-Mead (reflection / expansion / contraction / shrink) that asks for the objective in batches: the initial
    simplex at once, then reflection, expansion and both contractions of every step together (one pass of the bunch)."""
    n = len(x0)
    sim = np.vstack([x0] + [x0 + step * np.eye(n)[i] for i in range(n)])
    fv = f_batch(sim)
    evals = len(sim)
    for _ in range(iters):
        order = np.argsort(fv)
        sim, fv = sim[order], fv[order]
        c = sim[:-1].mean(axis=0)
        cand = np.vstack([c + (c - sim[-1]), c + 2.0 * (c - sim[-1]), c + 0.5 * (c - sim[-1]), c - 0.5 * (c - sim[-1])])
        fr, fe, foc, fic = f_batch(cand)
        evals += 4
        if fr < fv[0]:
            sim[-1], fv[-1] = (cand[1], fe) if fe < fr else (cand[0], fr)
        elif fr < fv[-2]:
            sim[-1], fv[-1] = cand[0], fr
        elif fr < fv[-1] and foc <= fr:
            sim[-1], fv[-1] = cand[2], foc
        elif fic < fv[-1]:
            sim[-1], fv[-1] = cand[3], fic
        else:
            sim[1:] = sim[0] + 0.5 * (sim[1:] - sim[0])
            fv[1:] = f_batch(sim[1:])
            evals += n
    best = int(np.argmin(fv))
    return sim[best], float(fv[best]), evals


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--stages", type=int, default=15)
    ap.add_argument("--n", type=int, default=1_000_000)
    args = ap.parse_args()
    import torch
    import paper_2402_17248_b200 as hb
    hb.lib()
    g = [1.0 + 1000.0 / wl.ELECTRON_MEV + j * 7000.0 / wl.ELECTRON_MEV for j in range(args.stages + 1)]
    bg = [math.sqrt(v * v - 1.0) for v in g]
    s = wl.NOMINAL_SIGMA
    sd = np.array([s[0], s[2], s[4], bg[0] * s[1], bg[0] * s[3], bg[0] * s[5]])
    coords = hb.to_device(wl.gaussian_bunch(args.n, 15))
    params, total_evals, t_eval = [], 0, 0.0
    for j in range(args.stages):
        kin_in = (g[j] - 1.0) * wl.ELECTRON_MEV
        kin_out = (g[j + 1] - 1.0) * wl.ELECTRON_MEV
        stage = hb.Lattice.from_description(wl.lattice([stage_description(j, bg[j], bg[j + 1], sd)], kin_in), device=0)
        stage.push(coords)
        stage.close()
        if j == args.stages - 1:
            break
        gap = hb.Lattice.from_description(wl.lattice(gap_description(0.5, 0.0), kin_out), device=0)
        spx = s[1] * bg[0] / bg[j + 1]                        # nominal divergence at this energy

        def objective(batch):
            nonlocal t_eval
            d = np.clip(batch[:, 0], 0.02, 0.98)
            length = np.stack([d, np.full(len(d), 0.05), 1.0 - d], axis=1)
            param = np.stack([np.zeros(len(d)), batch[:, 1], np.zeros(len(d))], axis=1)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            rec = gap.push_candidates(coords, [0, 1, 2], length, param).cpu().numpy()
            t_eval += time.perf_counter() - t0
            # C_xx / sx^2 + C_pxpx / spx^2 + C_yy / sy^2 + C_pypy / spy^2 behind the gap (record layout of hb_push_moments)
            return rec[:, 6] / s[0] ** 2 + rec[:, 12] / spx ** 2 + rec[:, 17] / s[2] ** 2 + rec[:, 21] / spx ** 2

        best, fbest, evals = nelder_mead_batched(objective, np.array([0.5, 1.0]), np.array([0.1, 1.0]))
        total_evals += evals
        d = float(np.clip(best[0], 0.02, 0.98))
        for idx, (L, p) in enumerate(((d, 0.0), (0.05, best[1]), (1.0 - d, 0.0))):
            gap.set_element(idx, L, p)
        rec = gap.push_moments(coords).cpu().numpy()[0]
        gap.close()
        params.append((d, float(best[1])))
        print("gap %2d: lens at %.3f m, k = %+8.3f m^-2 -> sigma_x = %.3e m, sigma_y = %.3e m (%d evaluations)" %
              (j + 1, d, best[1], math.sqrt(rec[6]), math.sqrt(rec[17]), evals))
    torch.cuda.synchronize()
    print("%d parameters over %d gaps, %d objective evaluations on a %d-particle bunch: %.1f evaluations/s "
          "(%.2f ms per evaluation incl. the host round trip)" %
          (2 * len(params), len(params), total_evals, args.n, total_evals / max(t_eval, 1e-9), 1e3 * t_eval / max(total_evals, 1)))


if __name__ == "__main__":
    main()
