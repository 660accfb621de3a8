"""Seeded synthetic workloads C1..C5 (BASELINE.json `configs`).

This module only *describes* inputs: particle arrays, network weights, normalisation
constants and lattice element lists, as plain Python/numpy data.  It holds none of the
method's arithmetic (no element map, no MLP evaluation, no moments, no s<->t conversion)
and imports neither `oracle/` nor the CUDA package; both consume the same description.

Lattice description = dict(kinetic_MeV, rest_MeV, elements=[...]) with elements
  {"kind": "drift", "L": m}
  {"kind": "quad", "L": m, "k": 1/m^2}            (k > 0 focuses x)
  {"kind": "sbend", "L": m, "theta": rad}
  {"kind": "monitor"}
  {"kind": "surrogate", "widths": [6,H,..,H,6], "W": [f32 (out,in) ...], "b": [f32 ...],
   "act": "identity"|"relu"|"prelu"|"tanh", "prelu_a": f32[n_hidden] | None,
   "in_mean","in_std","out_mean","out_std": f64[6], "coord": "s"|"t",
   "ref_bg_out": float (NaN = derive), "ref_z_out": float (NaN = derive), "prec": str}

Random numbers: numpy default_rng (PCG64); particles from default_rng([seed, 0]), the
network of stage j from default_rng([seed, 1, j]); seed = config number.  Values are drawn
in fp64, scaled, and rounded to fp32; the fp32 values are the common input of the oracle
and of the CUDA path.  The paper's own particle data and trained weights (Zenodo)
are not available; these stand in for them with the paper's shapes (P:156, P:164-169,
P:177).
"""
from __future__ import annotations

import math
import numpy as np

ELECTRON_MEV = 0.51099895
COORDS = ("x", "px", "y", "py", "t", "pt")
# BASELINE.json config 1: rms sizes of the uncorrelated Gaussian bunch, SoA order
NOMINAL_SIGMA = np.array([1e-3, 1e-4, 1e-3, 1e-4, 1e-3, 1e-3], dtype=np.float64)


# ----------------------------------------------------------------------------- particles
def gaussian_bunch(n: int, seed: int, sigma=NOMINAL_SIGMA, chunk: int = 1 << 22) -> np.ndarray:
    """[6, n] float32, independent N(0, sigma_j^2) per coordinate."""
    rng = np.random.default_rng([seed, 0])
    out = np.empty((6, n), dtype=np.float32)
    for s in range(0, n, chunk):
        e = min(n, s + chunk)
        z = rng.standard_normal((6, e - s))
        out[:, s:e] = (z * np.asarray(sigma, dtype=np.float64)[:, None]).astype(np.float32)
    return out


def correlated_bunch(n: int, seed: int, chunk: int = 1 << 22) -> np.ndarray:
    """[6, n] float32 correlated Gaussian: G iid N(0,1) 6x6, Sigma = G G^T, X = chol(Sigma) Z."""
    rng = np.random.default_rng([seed, 0])
    g = rng.standard_normal((6, 6))
    chol = np.linalg.cholesky(g @ g.T)
    out = np.empty((6, n), dtype=np.float32)
    for s in range(0, n, chunk):
        e = min(n, s + chunk)
        out[:, s:e] = (chol @ rng.standard_normal((6, e - s))).astype(np.float32)
    return out


# ------------------------------------------------------------------------------ networks
def make_mlp(widths, init: str, seed: int, stage: int):
    """Weights (row-major [out][in]) and biases as float32 lists.
    init 'xavier': U(-a, a), a = sqrt(6/(fan_in+fan_out)); 'he': N(0, 2/fan_in).
    Biases U(-1/sqrt(fan_in), +1/sqrt(fan_in)) (G15)."""
    rng = np.random.default_rng([seed, 1, stage])
    W, b = [], []
    for fin, fout in zip(widths[:-1], widths[1:]):
        if init == "xavier":
            a = math.sqrt(6.0 / (fin + fout))
            w = rng.uniform(-a, a, size=(fout, fin))
        elif init == "he":
            w = rng.standard_normal((fout, fin)) * math.sqrt(2.0 / fin)
        else:
            raise ValueError(init)
        bb = rng.uniform(-1.0 / math.sqrt(fin), 1.0 / math.sqrt(fin), size=(fout,))
        W.append(np.ascontiguousarray(w, dtype=np.float32))
        b.append(np.ascontiguousarray(bb, dtype=np.float32))
    return W, b


def surrogate(widths, W, b, act, in_mean, in_std, out_mean, out_std, coord="s",
              prelu_a=None, ref_bg_out=float("nan"), ref_z_out=float("nan"), prec="fp32"):
    return {
        "kind": "surrogate", "widths": [int(w) for w in widths], "W": W, "b": b, "act": act,
        "prelu_a": None if prelu_a is None else np.asarray(prelu_a, dtype=np.float32),
        "in_mean": np.asarray(in_mean, dtype=np.float64), "in_std": np.asarray(in_std, dtype=np.float64),
        "out_mean": np.asarray(out_mean, dtype=np.float64), "out_std": np.asarray(out_std, dtype=np.float64),
        "coord": coord, "ref_bg_out": float(ref_bg_out), "ref_z_out": float(ref_z_out), "prec": prec,
    }


# ------------------------------------------------------------------------------ lattices
def drift(L): return {"kind": "drift", "L": float(L)}
def drift_exact(L): return {"kind": "drift_exact", "L": float(L)}
def quad_chromatic(L, k): return {"kind": "quad_chromatic", "L": float(L), "k": float(k)}
def multipole(order, kn, ks=0.0): return {"kind": "multipole", "order": int(order), "kn": float(kn), "ks": float(ks)}
def quad(L, k): return {"kind": "quad", "L": float(L), "k": float(k)}
def sbend(L, theta): return {"kind": "sbend", "L": float(L), "theta": float(theta)}
def plens(L, k): return {"kind": "plens", "L": float(L), "k": float(k)}
def monitor(): return {"kind": "monitor"}


def fodo_cell(k):
    return [drift(0.25), quad(0.1, +k), drift(0.5), quad(0.1, -k), drift(0.25)]


def lattice(elements, kinetic_MeV=1000.0, rest_MeV=ELECTRON_MEV):
    return {"kinetic_MeV": float(kinetic_MeV), "rest_MeV": float(rest_MeV), "elements": list(elements)}


def config1(prec="fp32", n=4096):
    """PR1 ref: FODO cell (k=1) | surrogate 6-64-64-6 tanh Xavier, COORD_S | drift 0.25; monitor after each."""
    W, b = make_mlp([6, 64, 64, 6], "xavier", 1, 0)
    zero = np.zeros(6)
    el = fodo_cell(1.0) + [monitor(),
                           surrogate([6, 64, 64, 6], W, b, "tanh", zero, NOMINAL_SIGMA, zero, NOMINAL_SIGMA, prec=prec),
                           monitor(), drift(0.25), monitor()]
    return lattice(el), gaussian_bunch(n, 1)


def config2(n=1_000_000, cells=100):
    """Conventional only: `cells` FODO cells with k=1.2 (one run of 5*cells elements), one monitor."""
    el = []
    for _ in range(cells):
        el += fodo_cell(1.2)
    el.append(monitor())
    return lattice(el), gaussian_bunch(n, 2)


def config3(prec="bf16", n=10_000_000, widths=(6, 256, 256, 256, 6), act="relu", init="he",
            with_monitor=True, prelu_a=None):
    """Surrogate only: correlated Gaussian bunch, 6-256^3-6 ReLU He, mean/std input normalisation."""
    x = correlated_bunch(n, 3)
    x64 = x.astype(np.float64)
    mu, sd = x64.mean(axis=1), x64.std(axis=1)
    W, b = make_mlp(list(widths), init, 3, 0)
    el = [surrogate(list(widths), W, b, act, mu, sd, np.zeros(6), np.ones(6), prec=prec, prelu_a=prelu_a)]
    if with_monitor:
        el.append(monitor())
    return lattice(el), x


def c4_transport():
    el = [drift(0.25), quad(0.1, +1.2), drift(0.5), quad(0.1, -1.2), drift(0.5),
          quad(0.1, +1.2), drift(0.5), quad(0.1, -1.2), drift(0.25)]
    el += [sbend(0.5, +0.02), sbend(0.5, -0.02), sbend(0.5, -0.02), sbend(0.5, +0.02)]
    return el


def config4(prec="bf16", n=10_000_000, stages=2, gain_MeV=7000.0):
    """Hybrid: [surrogate COORD_T 6-128^3-6 tanh Xavier; 4 quads + 5 drifts + 4-sbend chicane] x stages,
    monitor after each segment; +7 GeV reference energy per stage."""
    g = [1.0 + 1000.0 / ELECTRON_MEV]
    for _ in range(stages):
        g.append(g[-1] + gain_MeV / ELECTRON_MEV)
    bg = [math.sqrt(gg * gg - 1.0) for gg in g]
    b0 = bg[0] / g[0]
    s = NOMINAL_SIGMA
    sd = np.array([s[0], s[2], b0 * s[4], bg[0] * s[1], bg[0] * s[3], bg[0] * s[5] / b0])
    el = []
    for j in range(stages):
        W, b = make_mlp([6, 128, 128, 128, 6], "xavier", 4, j)
        mu_in = np.array([0, 0, 0, 0, 0, bg[j]], dtype=np.float64)
        mu_out = np.array([0, 0, 0, 0, 0, bg[j + 1]], dtype=np.float64)
        el.append(surrogate([6, 128, 128, 128, 6], W, b, "tanh", mu_in, sd, mu_out, sd, coord="t",
                            ref_bg_out=bg[j + 1], ref_z_out=0.0, prec=prec))
        el.append(monitor())
        el += c4_transport()
        el.append(monitor())
    return lattice(el), gaussian_bunch(n, 4)


def config5(prec="bf16", n=100_000_000, stages=9, width=512, particles=True):
    """Large bunch: 9 surrogates COORD_S 6-512^4-6 tanh Xavier, interleaved with 8 runs of 10 FODO cells."""
    zero = np.zeros(6)
    widths = [6] + [width] * 4 + [6]
    el = []
    for j in range(stages):
        W, b = make_mlp(widths, "xavier", 5, j)
        el.append(surrogate(widths, W, b, "tanh", zero, NOMINAL_SIGMA, zero, NOMINAL_SIGMA, prec=prec))
        el.append(monitor())
        if j < stages - 1:
            for _ in range(10):
                el += fodo_cell(1.2)
            el.append(monitor())
    return lattice(el), (gaussian_bunch(n, 5) if particles else None)


def paper_net(width, hidden, prec="bf16", n=10_000_000, particles=True):
    """One stage with the paper's own network shape (5 hidden x 900 for stages 1-3, 3 hidden x 700 for stages
    4-15, PReLU), He-initialised weights from the seed (the trained weights are not available), COORD_S, N = 1e7 as
    in the paper's timing; monitor after the stage."""
    zero = np.zeros(6)
    widths = [6] + [int(width)] * int(hidden) + [6]
    W, b = make_mlp(widths, "he", 7, int(width))
    a = np.full(len(widths) - 2, 0.25, dtype=np.float32)       # PyTorch's default PReLU slope
    el = [surrogate(widths, W, b, "prelu", zero, NOMINAL_SIGMA, zero, NOMINAL_SIGMA, prelu_a=a, prec=prec), monitor()]
    return lattice(el), (gaussian_bunch(n, 7) if particles else None)


def subsample_indices(n: int, m: int = 1 << 20) -> np.ndarray:
    """Fixed parity subsample: every floor(n/m)-th particle, m particles (all of them if n <= m)."""
    if n <= m:
        return np.arange(n)
    return np.arange(m) * (n // m)


def flops_per_particle(widths) -> int:
    return 2 * sum(a * b for a, b in zip(widths[:-1], widths[1:]))


def shard_range(n: int, rank: int, world: int):
    """Contiguous particle range of `rank` (DESIGN.md multi-GPU: particles shard, nothing else moves)."""
    base, rem = divmod(n, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)
