"""Pins of the fp64 oracle against what the mathematics fixes (CPU only).

Nothing here re-types the oracle's formulas and calls that a check: each test uses a closed
form, an invariant, a limit, a brute-force numpy evaluation with a different structure, or a
value stored in tests/golden/survey_pins.txt (computed outside oracle/).  DESIGN.md lists the
readings R1-R10 these pin.
"""
import math
import os

import numpy as np
import pytest

import oracle
import workloads as wl

MC2 = wl.ELECTRON_MEV
GOLD = {}
with open(os.path.join(os.path.dirname(__file__), "golden", "survey_pins.txt")) as f:
    for line in f:
        if line.strip() and not line.startswith("#"):
            k, v = line.split()
            GOLD[k] = float(v)

G0, BG0, B0 = oracle.reference(1000.0, MC2)
S6 = np.kron(np.eye(3), np.array([[0.0, 1.0], [-1.0, 0.0]]))
LAT = wl.lattice([])


def jacobian(elements, bg=None):
    """6x6 matrix of a list of (linear) elements: push the 6 unit vectors and the origin."""
    c = np.zeros((6, 7))
    c[:, :6] = np.eye(6)
    tr = oracle.Tracker(LAT)
    if bg is not None:
        tr.bg = bg
    for el in elements:
        tr.apply(el, c)
    assert np.all(c[:, 6] == 0.0)          # linear maps keep the origin
    return c[:, :6].copy()


def rand_coords(n, seed=0, scale=wl.NOMINAL_SIGMA):
    rng = np.random.default_rng(seed)
    return np.ascontiguousarray(rng.standard_normal((6, n)) * scale[:, None])


# ------------------------------------------------------------------------------ R1
def test_reference_constants():
    assert G0 == pytest.approx(GOLD["gamma0"], rel=1e-15)
    assert BG0 == pytest.approx(GOLD["bg0"], rel=1e-14)
    assert B0 == pytest.approx(GOLD["beta0"], rel=1e-15)
    assert 1.0 / BG0 ** 2 == pytest.approx(GOLD["inv_bg0_sq"], rel=1e-12)
    assert G0 == 1.0 + 1000.0 / MC2 and abs(G0 * G0 - BG0 * BG0 - 1.0) < 1e-9


# ------------------------------------------------------------------------------ R2 drift
def test_drift_forward_backward_identity():
    c = rand_coords(1000)
    c0 = c.copy()
    oracle.drift(c, 0.37, BG0)
    assert not np.array_equal(c, c0)
    oracle.drift(c, -0.37, BG0)
    for j in (1, 3, 5):
        assert np.array_equal(c[j], c0[j])               # momenta untouched: bit exact
    for j in (0, 2, 4):
        assert np.max(np.abs(c[j] - c0[j])) <= 2 * np.spacing(np.max(np.abs(c0[j])))


def test_drift_matrix():
    L = 0.8
    M = jacobian([wl.drift(L)])
    E = np.eye(6)
    E[0, 1] = L
    E[2, 3] = L
    E[4, 5] = L / BG0 ** 2
    assert np.allclose(M, E, rtol=0, atol=1e-16)


def test_drift_t_slope_is_first_order_of_exact_kinematics():
    # c dt/ds - 1/beta0 for a particle with energy deviation pt (px=py=0), expanded to first order;
    # evaluated in 60-digit decimal arithmetic (the difference cancels 14 digits)
    from decimal import Decimal, getcontext
    getcontext().prec = 60
    g = Decimal(1) + Decimal(1000) / Decimal(repr(MC2))
    bg = (g * g - 1).sqrt()
    b0 = bg / g
    pt = Decimal("1e-9")
    exact = (1 / b0 - pt) / (1 - 2 * pt / b0 + pt * pt).sqrt() - 1 / b0
    assert float(exact / pt) == pytest.approx(1.0 / BG0 ** 2, rel=1e-5)
    M = jacobian([wl.drift(1.0)])
    assert M[4, 5] == pytest.approx(float(exact / pt), rel=1e-5)


# ------------------------------------------------------------------------------ R3 quad
@pytest.mark.parametrize("k", [1.2, -1.2, 0.3, -7.0])
def test_quad_matrix_closed_form(k):
    L = 0.1
    M = jacobian([wl.quad(L, k)])
    w = math.sqrt(abs(k))
    foc = np.array([[math.cos(w * L), math.sin(w * L) / w], [-w * math.sin(w * L), math.cos(w * L)]])
    dfc = np.array([[math.cosh(w * L), math.sinh(w * L) / w], [w * math.sinh(w * L), math.cosh(w * L)]])
    E = np.eye(6)
    E[0:2, 0:2] = foc if k > 0 else dfc
    E[2:4, 2:4] = dfc if k > 0 else foc
    E[4, 5] = L / BG0 ** 2
    assert np.allclose(M, E, rtol=0, atol=1e-15)
    assert abs(np.linalg.det(M[0:2, 0:2]) - 1) < 1e-14 and abs(np.linalg.det(M[2:4, 2:4]) - 1) < 1e-14


def test_quad_focuses_x_for_positive_k():
    M = jacobian([wl.quad(0.1, 1.0)])
    assert M[1, 0] < 0 < M[3, 2]


def test_quad_zero_strength_is_drift_and_limit():
    assert np.array_equal(jacobian([wl.quad(0.3, 0.0)]), jacobian([wl.drift(0.3)]))
    assert np.allclose(jacobian([wl.quad(0.3, 1e-12)]), jacobian([wl.drift(0.3)]), atol=1e-12)


def test_quad_inverse():
    M = jacobian([wl.quad(0.1, 1.2), wl.quad(-0.1, 1.2)])
    assert np.allclose(M, np.eye(6), atol=1e-15)


# ------------------------------------------------------------------------------ R4 sbend
def test_sbend_golden_values():
    M = jacobian([wl.sbend(0.5, 0.02)])
    idx = {"R11": (0, 0), "R12": (0, 1), "R21": (1, 0), "R16": (0, 5), "R26": (1, 5), "R51": (4, 0),
           "R52": (4, 1), "R56": (4, 5), "R34": (2, 3)}
    for name, (i, j) in idx.items():
        assert M[i, j] == pytest.approx(GOLD["sbend_" + name], rel=1e-12), name
    assert M[1, 1] == pytest.approx(GOLD["sbend_R11"], rel=1e-12)
    for i, j in [(0, 2), (0, 3), (0, 4), (2, 0), (2, 5), (3, 2), (5, 0), (5, 1), (5, 4), (4, 2)]:
        assert M[i, j] == 0.0
    assert M[5, 5] == 1.0 and M[4, 4] == 1.0 and M[2, 2] == 1.0 and M[3, 3] == 1.0


def test_sbend_dispersion_closed_form():
    # textbook sector dipole: R16 = rho (1 - cos theta) in delta=dp/p; here pt = -dE/(p0 c) so
    # dp/p = -pt/beta0 to first order  =>  d x / d pt = -rho (1-cos theta)/beta0
    L, th = 0.7, 0.05
    M = jacobian([wl.sbend(L, th)])
    rho = L / th
    assert M[0, 5] == pytest.approx(-rho * (1 - math.cos(th)) / B0, rel=1e-13)
    assert M[0, 1] == pytest.approx(rho * math.sin(th), rel=1e-13)
    assert M[1, 0] == pytest.approx(-math.sin(th) / rho, rel=1e-13)


def test_sbend_small_angle_limit_is_drift():
    D = jacobian([wl.drift(0.5)])
    assert np.array_equal(jacobian([wl.sbend(0.5, 0.0)]), D)
    assert np.allclose(jacobian([wl.sbend(0.5, 1e-9)]), D, atol=2e-9)
    # R56 -> L/(beta0 gamma0)^2 needs a cancellation-free comparison
    M = jacobian([wl.sbend(0.5, 1e-4)])
    assert M[4, 5] == pytest.approx(0.5 / BG0 ** 2 - 0.5 * 1e-8 / 6 / B0 ** 2, rel=1e-6)


def test_sbend_inverse_and_sign_symmetry():
    M = jacobian([wl.sbend(0.5, 0.02), wl.sbend(-0.5, -0.02)])
    assert np.allclose(M, np.eye(6), atol=1e-14)
    Mp, Mm = jacobian([wl.sbend(0.5, 0.02)]), jacobian([wl.sbend(0.5, -0.02)])
    F = np.diag([-1.0, -1.0, 1, 1, 1, 1])                 # mirror x
    assert np.allclose(F @ Mp @ F, Mm, atol=1e-16)


# ------------------------------------------------------------------------------ symplecticity
@pytest.mark.parametrize("els", [
    [wl.drift(0.4)], [wl.quad(0.1, 1.2)], [wl.quad(0.1, -1.2)], [wl.sbend(0.5, 0.02)], [wl.sbend(0.5, -0.3)],
    wl.fodo_cell(1.2), wl.c4_transport(), wl.fodo_cell(1.0) * 7 + wl.c4_transport(),
])
def test_symplectic(els):
    M = jacobian(els)
    assert np.max(np.abs(M.T @ S6 @ M - S6)) < 5e-15 * max(1.0, np.max(np.abs(M)) ** 2)


# ------------------------------------------------------------------------------ runs
def _block_params(M2):
    cmu = 0.5 * np.trace(M2)
    mu = math.acos(cmu)
    J = (M2 - np.eye(2) * cmu) / math.sin(mu)
    return mu, J


def test_fodo_cell_golden_and_de_moivre():
    M = jacobian(wl.fodo_cell(1.2))
    assert M[0, 0] == pytest.approx(GOLD["c2cell_x11"], rel=1e-13)
    assert M[0, 1] == pytest.approx(GOLD["c2cell_x12"], rel=1e-13)
    assert M[1, 0] == pytest.approx(GOLD["c2cell_x21"], rel=1e-12)
    assert M[1, 1] == pytest.approx(GOLD["c2cell_x22"], rel=1e-13)
    assert M[2, 2] == pytest.approx(GOLD["c2cell_x22"], rel=1e-13)     # y block: diagonal swapped
    assert M[3, 3] == pytest.approx(GOLD["c2cell_x11"], rel=1e-13)
    assert M[4, 5] == pytest.approx(GOLD["c2cell_R56"], rel=1e-12)
    mu, J = _block_params(M[0:2, 0:2])
    assert mu == pytest.approx(GOLD["c2cell_mu"], rel=1e-11)
    # 100 cells pushed element by element (500 oracle calls) vs De Moivre closed form
    M100 = jacobian(wl.fodo_cell(1.2) * 100)
    closed = np.eye(2) * math.cos(100 * mu) + J * math.sin(100 * mu)
    assert np.allclose(M100[0:2, 0:2], closed, rtol=0, atol=5e-11)
    assert M100[0, 0] == pytest.approx(GOLD["c2x100_x11"], rel=1e-10)
    assert M100[0, 1] == pytest.approx(GOLD["c2x100_x12"], rel=1e-10)
    assert M100[1, 0] == pytest.approx(GOLD["c2x100_x21"], rel=1e-10)
    assert M100[1, 1] == pytest.approx(GOLD["c2x100_x22"], rel=1e-10)
    assert M100[4, 5] == pytest.approx(GOLD["c2x100_R56"], rel=1e-11)
    assert M100[4, 5] == pytest.approx(100 * 1.2 / BG0 ** 2, rel=1e-12)   # R56 adds up: total length 120 m


def test_c1_cell_golden():
    M = jacobian(wl.fodo_cell(1.0))
    for n, (i, j) in {"x11": (0, 0), "x12": (0, 1), "x21": (1, 0), "x22": (1, 1)}.items():
        assert M[i, j] == pytest.approx(GOLD["c1cell_" + n], rel=1e-12)


def test_c4_transport_golden():
    M = jacobian(wl.c4_transport())
    idx = {"R11": (0, 0), "R12": (0, 1), "R21": (1, 0), "R22": (1, 1), "R16": (0, 5), "R26": (1, 5),
           "R33": (2, 2), "R34": (2, 3), "R43": (3, 2), "R44": (3, 3), "R51": (4, 0), "R52": (4, 1), "R56": (4, 5)}
    for name, (i, j) in idx.items():
        assert M[i, j] == pytest.approx(GOLD["c4_" + name], rel=2e-6), name


def test_run_equals_product_of_matrices_on_8_particles():
    els = wl.fodo_cell(1.2) + wl.c4_transport() + [wl.quad(0.2, -0.7), wl.sbend(0.3, -0.1)]
    P = np.eye(6)
    for el in els:
        P = jacobian([el]) @ P
    c0 = rand_coords(8, seed=5)
    c, _ = oracle.push(wl.lattice(els), c0)
    assert np.allclose(c, P @ c0, rtol=1e-13, atol=1e-20)


def test_element_order_matters_and_is_lattice_order():
    a, b = [wl.quad(0.1, 3.0), wl.drift(1.0)], [wl.drift(1.0), wl.quad(0.1, 3.0)]
    Ma, Mb = jacobian(a), jacobian(b)
    assert not np.allclose(Ma, Mb)
    assert np.allclose(Ma, jacobian([a[1]]) @ jacobian([a[0]]), atol=1e-15)


# ------------------------------------------------------------------------------ R10 moments
def test_moments_by_hand_8_particles():
    c = np.zeros((6, 8))
    c[0] = [1, 2, 3, 4, 5, 6, 7, 8]
    c[1] = [1, -1, 1, -1, 1, -1, 1, -1]
    c[5] = [2, 2, 2, 2, 4, 4, 4, 4]
    m = oracle.moments(c)
    assert m[0] == 4.5 and m[1] == 0.0 and m[5] == 3.0
    assert m[6] == pytest.approx(5.25)            # var(1..8), 1/N
    assert m[7] == pytest.approx(-0.5)            # cov(x, px)
    assert m[11] == pytest.approx(2.0)            # cov(x, pt) = mean((x-4.5)*(pt-3)) = (2.5+1.5+.5... )
    assert m[12] == pytest.approx(1.0)            # var(px)
    assert m[26] == pytest.approx(1.0)            # var(pt)
    assert m[2] == 0 and m[17] == 0               # y untouched


def test_moments_match_numpy_cov_population():
    c = rand_coords(5000, seed=3) + np.arange(6)[:, None] * 1e-3
    m = oracle.moments(c)
    C = np.cov(c, bias=True)
    iu = np.triu_indices(6)
    assert np.allclose(m[:6], c.mean(axis=1), rtol=1e-13)
    assert np.allclose(m[6:], C[iu], rtol=1e-11, atol=1e-22)


def emit(m, j):
    C = np.zeros((6, 6))
    C[np.triu_indices(6)] = m[6:]
    C = C + C.T - np.diag(np.diag(C))
    return math.sqrt(C[j, j] * C[j + 1, j + 1] - C[j, j + 1] ** 2), C


def test_covariance_transport_and_emittance_conservation():
    c0 = rand_coords(20000, seed=7)
    lat, _ = wl.config2(n=1, cells=100)
    M = jacobian(lat["elements"][:-1])
    m0 = oracle.moments(np.ascontiguousarray(c0))
    c1, rec = oracle.push(lat, c0)
    ex0, C0 = emit(m0, 0)
    ex1, C1 = emit(rec[0], 0)
    ey0, ey1 = emit(m0, 2)[0], emit(rec[0], 2)[0]
    assert abs(ex1 / ex0 - 1) < 1e-11 and abs(ey1 / ey0 - 1) < 1e-11       # uncoupled quad/drift run
    assert np.allclose(C1, M @ C0 @ M.T, rtol=1e-10, atol=1e-22)          # exact sample identity
    # chicane: eps_x leaks (dispersion) but det Sigma_6 is conserved
    lat4 = wl.lattice(wl.c4_transport() + [wl.monitor()])
    _, rec4 = oracle.push(lat4, c0)
    C4 = emit(rec4[0], 0)[1]
    s0, l0 = np.linalg.slogdet(C0)
    s4, l4 = np.linalg.slogdet(C4)
    assert s0 == s4 == 1 and abs(l4 - l0) < 1e-8


# ------------------------------------------------------------------------------ R6 s<->t
def test_s_t_round_trip_identity():
    c = rand_coords(4096, seed=11)
    back = oracle.to_s(oracle.to_t(c, BG0), BG0)
    err = np.max(np.abs(back - c), axis=1) / wl.NOMINAL_SIGMA
    assert np.max(err) < 1e-12


def test_to_t_reference_particle_and_first_order_limits():
    c = np.zeros((6, 1))
    v = oracle.to_t(c, BG0)
    assert np.array_equal(v[:5, 0], np.zeros(5)) and v[5, 0] == pytest.approx(BG0, rel=1e-15)
    eps = 1e-7
    c = np.zeros((6, 2))
    c[4, 0] = eps          # late particle: z_t -> -beta0 t
    c[5, 1] = eps          # energy deviation: uz - uz0 -> -pt (beta gamma)0 / beta0
    v = oracle.to_t(c, BG0)
    assert v[2, 0] / eps == pytest.approx(-B0, rel=1e-9)
    assert (v[5, 1] - BG0) / eps == pytest.approx(-BG0 / B0, rel=1e-5)
    # transverse: ux = px * bg0, and x_t = x - (ux/gamma) t
    c = np.zeros((6, 1))
    c[0, 0], c[1, 0], c[4, 0] = 1e-3, 2e-4, 5e-4
    v = oracle.to_t(c, BG0)
    assert v[3, 0] == pytest.approx(2e-4 * BG0, rel=1e-15)
    assert v[0, 0] == pytest.approx(1e-3 - (2e-4 * BG0 / G0) * 5e-4, rel=1e-14)


def test_to_s_energy_and_time_definitions():
    # a particle with momentum purely along z, gamma = g1 + dg, sitting dz ahead of the reference
    bg1 = 5000.0
    g1 = math.sqrt(1 + bg1 * bg1)
    dg, dz = 3.0, 2e-5
    uz = math.sqrt((g1 + dg) ** 2 - 1)
    v = np.array([[0.0], [0.0], [dz], [0.0], [0.0], [uz]])
    s = oracle.to_s(v, bg1)
    assert s[5, 0] == pytest.approx(-dg / bg1, rel=1e-9)                     # pt = -(gamma-g1)/(bg1)
    assert s[4, 0] == pytest.approx(-dz * (g1 + dg) / uz, rel=1e-14)         # ahead => early (t<0)
    assert s[4, 0] < 0


# ------------------------------------------------------------------------------ R8/R9 MLP
def _sur(widths, W, b, act, prelu_a=None, **kw):
    z, o = np.zeros(6), np.ones(6)
    d = dict(in_mean=z, in_std=o, out_mean=z, out_std=o)
    d.update(kw)
    return wl.surrogate(widths, W, b, act, d["in_mean"], d["in_std"], d["out_mean"], d["out_std"],
                        prelu_a=prelu_a)


def test_identity_initialised_prelu():
    H = 10
    A0 = np.zeros((H, 6), np.float32); A0[:6] = np.eye(6)
    A1 = np.zeros((H, H), np.float32); A1[:6, :6] = np.eye(6)
    A2 = np.zeros((6, H), np.float32); A2[:, :6] = np.eye(6)
    zb = [np.zeros(H, np.float32), np.zeros(H, np.float32), np.zeros(6, np.float32)]
    sur = _sur([6, H, H, 6], [A0, A1, A2], zb, "prelu", prelu_a=[1.0, 1.0])
    c = rand_coords(100, seed=2, scale=np.ones(6))
    c0 = c.copy()
    oracle.mlp_normalised(c, sur)
    assert np.array_equal(c, c0)


def test_identity_via_relu_pair():
    H = 12
    A0 = np.zeros((H, 6), np.float32); A0[:6] = np.eye(6); A0[6:12] = -np.eye(6)
    A1 = np.zeros((6, H), np.float32); A1[:, :6] = np.eye(6); A1[:, 6:12] = -np.eye(6)
    sur = _sur([6, H, 6], [A0, A1], [np.zeros(H, np.float32), np.zeros(6, np.float32)], "relu")
    c = rand_coords(100, seed=4, scale=np.ones(6))
    c0 = c.copy()
    oracle.mlp_normalised(c, sur)
    assert np.array_equal(c, c0)          # z = relu(z) - relu(-z)


def test_relu_and_prelu_pointwise_definition():
    # 6 -> 6 -> 6 with identity matrices: output = act(input) (Eq. 1, Eq. 2)
    I = np.eye(6, dtype=np.float32)
    zb = [np.zeros(6, np.float32)] * 2
    c = np.array([[-2.0, -0.5, 0.0, 0.5, 2.0]] * 6)
    for act, a, f in [("relu", None, lambda z: np.where(z >= 0, z, 0.0)),
                      ("prelu", [0.25], lambda z: np.where(z >= 0, z, 0.25 * z)),
                      ("tanh", None, np.tanh), ("identity", None, lambda z: z)]:
        v = c.copy()
        oracle.mlp_normalised(v, _sur([6, 6, 6], [I, I], zb, act, prelu_a=a))
        assert np.allclose(v, f(c), rtol=1e-15, atol=0), act


@pytest.mark.parametrize("act", ["tanh", "relu", "prelu"])
def test_mlp_brute_force_8_particles(act):
    widths = [6, 17, 9, 6]
    W, b = wl.make_mlp(widths, "xavier", 99, 0)
    rng = np.random.default_rng(1)
    stats = dict(in_mean=rng.normal(size=6), in_std=rng.uniform(0.5, 2, 6),
                 out_mean=rng.normal(size=6), out_std=rng.uniform(0.5, 2, 6))
    a = [0.125, 0.3125] if act == "prelu" else None      # exactly representable in fp32
    sur = _sur(widths, W, b, act, prelu_a=a, **stats)
    c = rand_coords(8, seed=8, scale=np.ones(6))
    # dense numpy evaluation, batch-major (structurally different from the per-particle loops)
    h = ((c - stats["in_mean"][:, None]) / stats["in_std"][:, None]).T
    for l in range(3):
        h = h @ W[l].astype(np.float64).T + b[l].astype(np.float64)
        if l < 2:
            if act == "tanh":
                h = np.vectorize(math.tanh)(h)
            elif act == "relu":
                h = np.maximum(h, 0)
            else:
                h = np.where(h >= 0, h, a[l] * h)
    expect = h.T * stats["out_std"][:, None] + stats["out_mean"][:, None]
    oracle.mlp_normalised(c, sur)
    assert np.allclose(c, expect, rtol=1e-13, atol=1e-15)


def test_identity_activation_is_single_affine_map():
    widths = [6, 20, 20, 6]
    W, b = wl.make_mlp(widths, "he", 7, 0)
    sur = _sur(widths, W, b, "identity")
    A = np.eye(6)
    off = np.zeros(6)
    for l in range(3):
        A = W[l].astype(np.float64) @ A
        off = W[l].astype(np.float64) @ off + b[l]
    c = rand_coords(50, seed=9, scale=np.ones(6))
    expect = A @ c + off[:, None]
    oracle.mlp_normalised(c, sur)
    assert np.allclose(c, expect, rtol=1e-12, atol=1e-14)


def test_tanh_net_is_odd_without_biases():
    widths = [6, 16, 16, 6]
    W, b = wl.make_mlp(widths, "xavier", 5, 0)
    sur = _sur(widths, W, [np.zeros_like(x) for x in b], "tanh")
    c = rand_coords(64, seed=10, scale=np.ones(6))
    m = -c
    oracle.mlp_normalised(c, sur)
    oracle.mlp_normalised(m, sur)
    assert np.array_equal(c, -m)


def test_cross_pin_linear_surrogate_reproduces_element_matrix():
    # a 1-layer identity-activation COORD_S surrogate with A = D_out^-1 M D_in reproduces element M
    M = jacobian(wl.fodo_cell(1.2))
    sd = wl.NOMINAL_SIGMA
    A = (np.diag(1 / sd) @ M @ np.diag(sd)).astype(np.float32)
    sur = wl.surrogate([6, 6], [A], [np.zeros(6, np.float32)], "identity", np.zeros(6), sd, np.zeros(6), sd)
    c0 = rand_coords(256, seed=12)
    c = c0.copy()
    oracle.mlp_normalised(c, sur)
    assert np.max(np.abs(c - M @ c0) / sd[:, None]) < 1e-6      # fp32 rounding of A only


# ------------------------------------------------------------------------------ R7 reference update
def test_reference_update_given_and_auto():
    widths = [6, 8, 6]
    W, b = wl.make_mlp(widths, "xavier", 3, 0)
    bgs = BG0 * 2
    sd = np.array([1e-3, 1e-3, 1e-3, 0.2, 0.2, 2.0])
    mu_in = np.array([0, 0, 0, 0, 0, BG0])
    mu_out = np.array([0, 0, 0, 0, 0, bgs])
    sur = wl.surrogate(widths, W, b, "tanh", mu_in, sd, mu_out, sd, coord="t", ref_bg_out=bgs, ref_z_out=0.0)
    # reference-identical particle: evaluate net on reference input by brute force numpy
    h = (np.array([0, 0, 0, 0, 0, BG0]) - mu_in) / sd
    h = np.tanh(W[0].astype(np.float64) @ h + b[0])
    r = (W[1].astype(np.float64) @ h + b[1]) * sd + mu_out
    g_out = math.sqrt(1 + r[3] ** 2 + r[4] ** 2 + r[5] ** 2)
    g1 = math.sqrt(1 + bgs ** 2)
    c, _ = oracle.push(wl.lattice([sur]), np.zeros((6, 1)))
    assert c[5, 0] == pytest.approx(-(g_out - g1) / bgs, rel=1e-10)
    assert c[1, 0] == pytest.approx(r[3] / bgs, rel=1e-12)
    # auto (NaN): reference comes out at t = 0 and pt = -(gamma(r)-gamma(uz only))/bg1
    sur2 = dict(sur, ref_bg_out=float("nan"), ref_z_out=float("nan"))
    c2, _ = oracle.push(wl.lattice([sur2]), np.zeros((6, 1)))
    assert c2[4, 0] == 0.0
    g1a = math.sqrt(1 + r[5] ** 2)
    assert c2[5, 0] == pytest.approx(-(g_out - g1a) / r[5], rel=1e-9, abs=1e-18)
    # downstream elements use the new reference: a drift after the stage has R56 = L/bg1^2
    tr = oracle.Tracker(wl.lattice([]))
    cc = np.zeros((6, 1))
    tr.apply(sur, cc)
    assert tr.bg == bgs
    cc[:] = 0
    cc[5, 0] = 1e-3
    tr.apply(wl.drift(2.0), cc)
    assert cc[4, 0] == pytest.approx(2.0 * 1e-3 / bgs ** 2, rel=1e-14)


def test_coord_s_surrogate_keeps_reference():
    lat, x = wl.config1(n=64)
    tr = oracle.Tracker(lat)
    c = np.ascontiguousarray(x.astype(np.float64))
    for el in lat["elements"]:
        tr.apply(el, c)
    assert tr.bg == BG0 and len(tr.records) == 3


def test_config4_physical_no_nans():
    lat, x = wl.config4(n=2048)
    c, rec = oracle.push(lat, x)
    assert np.all(np.isfinite(c)) and rec.shape == (4, 27) and np.all(np.isfinite(rec))


# ------------------------------------------------------------------------------ R3b plasma lens (NEXT-2)
@pytest.mark.parametrize("k", [3.0, -3.0, 250.0])
def test_plens_matrix_closed_form(k):
    """x'' = -k x in BOTH planes: the textbook harmonic-oscillator transfer matrix, twice; t as in a drift"""
    L = 0.05
    M = jacobian([wl.plens(L, k)])
    w = math.sqrt(abs(k))
    foc = np.array([[math.cos(w * L), math.sin(w * L) / w], [-w * math.sin(w * L), math.cos(w * L)]])
    dfc = np.array([[math.cosh(w * L), math.sinh(w * L) / w], [w * math.sinh(w * L), math.cosh(w * L)]])
    E = np.eye(6)
    E[0:2, 0:2] = E[2:4, 2:4] = foc if k > 0 else dfc
    E[4, 5] = L / BG0 ** 2
    assert np.allclose(M, E, rtol=0, atol=1e-14)
    assert np.max(np.abs(M.T @ S6 @ M - S6)) < 1e-13 * max(1.0, np.max(np.abs(M)) ** 2)


def test_plens_is_a_quad_in_x_and_the_opposite_quad_in_y():
    """cross pin against the (separately pinned) quadrupole: lens(k) = quad(+k) in x = quad(-k) in y"""
    L, k = 0.07, 11.0
    P, Qp, Qm = jacobian([wl.plens(L, k)]), jacobian([wl.quad(L, k)]), jacobian([wl.quad(L, -k)])
    assert np.array_equal(P[0:2, 0:2], Qp[0:2, 0:2]) and np.array_equal(P[2:4, 2:4], Qm[2:4, 2:4])
    assert np.array_equal(P[4:6, :], Qp[4:6, :])
    assert P[1, 0] < 0 and P[3, 2] < 0                       # focuses both planes for k > 0


def test_plens_limits_inverse_and_thin_lens():
    assert np.array_equal(jacobian([wl.plens(0.3, 0.0)]), jacobian([wl.drift(0.3)]))
    assert np.allclose(jacobian([wl.plens(0.02, 9.0), wl.plens(-0.02, 9.0)]), np.eye(6), atol=1e-15)
    # thin-lens limit: L -> 0 at fixed integrated strength kL = 1/f: kick px -= x/f, no displacement
    f, L = 2.0, 1e-7
    M = jacobian([wl.plens(L, 1.0 / (f * L))])
    assert abs(M[1, 0] + 1.0 / f) < 1e-6 and abs(M[0, 0] - 1.0) < 1e-6 and abs(M[0, 1]) < 1e-6
    # a quarter betatron period images (x, px) -> (px / w, -w x)
    w = 5.0
    M = jacobian([wl.plens(math.pi / (2 * w), w * w)])
    assert np.allclose(M[0:2, 0:2], [[0.0, 1.0 / w], [-w, 0.0]], atol=1e-15)


def test_plens_8_particles_brute_force_and_axisymmetry():
    c = rand_coords(8, 5)
    L, k = 0.05, 40.0
    ref = jacobian([wl.plens(L, k)]) @ c
    got = c.copy()
    oracle.Tracker(LAT).apply(wl.plens(L, k), got)
    assert np.allclose(got, ref, rtol=1e-13, atol=1e-20)
    # axisymmetric: rotating the transverse plane by any angle commutes with the lens (not true for a quadrupole)
    a = 0.7
    R = np.eye(6)
    R[np.ix_([0, 2], [0, 2])] = [[math.cos(a), -math.sin(a)], [math.sin(a), math.cos(a)]]
    R[np.ix_([1, 3], [1, 3])] = [[math.cos(a), -math.sin(a)], [math.sin(a), math.cos(a)]]
    P, Q = jacobian([wl.plens(L, k)]), jacobian([wl.quad(L, k)])
    assert np.allclose(R @ P, P @ R, atol=1e-14) and not np.allclose(R @ Q, Q @ R, atol=1e-3)


# ------------------------------------------------------------------------------ R2x exact drift (NEXT-3)
def test_exact_drift_is_straight_line_geometry_and_time_of_flight():
    """independent of the formula in the oracle: build the particle's velocity vector from (px, py, pt), fly it in a
    straight line until it has advanced by L in s, compare position and arrival time"""
    g0, bg0, b0 = oracle.reference(1000.0, wl.ELECTRON_MEV)[0], BG0, BG0 / math.sqrt(1 + BG0 ** 2)
    rng = np.random.default_rng(3)
    c = np.ascontiguousarray(rng.standard_normal((6, 64)) * np.array([1e-3, 2e-2, 1e-3, 2e-2, 1e-3, 5e-2])[:, None])
    L = 3.7
    got = c.copy()
    oracle.Tracker(LAT).apply(wl.drift_exact(L), got)
    for i in range(c.shape[1]):
        x, px, y, py, t, pt = c[:, i]
        gamma = g0 - pt * bg0                          # E = E0 - pt p0 c  (R1)
        p = math.sqrt(gamma ** 2 - 1.0) / bg0          # |p| / p0
        pz = math.sqrt(p * p - px * px - py * py)
        beta = math.sqrt(1.0 - 1.0 / gamma ** 2)
        path = L * p / pz                              # length of the straight line
        assert abs(got[0, i] - (x + path * px / p)) < 1e-14 and abs(got[2, i] - (y + path * py / p)) < 1e-14
        assert abs(got[4, i] - (t + path / beta - L / b0)) < 1e-12    # c (T - T_ref)
        assert got[1, i] == px and got[3, i] == py and got[5, i] == pt


def test_exact_drift_first_order_is_r2_and_it_is_symplectic():
    L = 0.9
    # Jacobian by central differences about the reference particle -> the matrix of R2
    h = 1e-6
    J = np.zeros((6, 6))
    for j in range(6):
        cp, cm = np.zeros((6, 1)), np.zeros((6, 1))
        cp[j], cm[j] = h, -h
        oracle.Tracker(LAT).apply(wl.drift_exact(L), cp)
        oracle.Tracker(LAT).apply(wl.drift_exact(L), cm)
        J[:, j] = (cp[:, 0] - cm[:, 0]) / (2 * h)
    assert np.allclose(J, jacobian([wl.drift(L)]), atol=1e-9)
    # ... and about a far-off-axis, off-momentum particle it is still a symplectic map
    c0 = np.array([2e-3, 3e-2, -1e-3, -2e-2, 5e-4, 4e-2])
    for j in range(6):
        cp, cm = c0.reshape(6, 1).copy(), c0.reshape(6, 1).copy()
        cp[j] += h; cm[j] -= h
        oracle.Tracker(LAT).apply(wl.drift_exact(L), cp)
        oracle.Tracker(LAT).apply(wl.drift_exact(L), cm)
        J[:, j] = (cp[:, 0] - cm[:, 0]) / (2 * h)
    assert np.max(np.abs(J.T @ S6 @ J - S6)) < 1e-8
    assert not np.allclose(J, jacobian([wl.drift(L)]), atol=1e-6)        # it does differ from R2 there


def test_exact_drift_composes_and_inverts():
    c = rand_coords(32, 9, scale=np.array([1e-3, 1e-2, 1e-3, 1e-2, 1e-3, 1e-2]))
    a, b = c.copy(), c.copy()
    tr = oracle.Tracker(LAT)
    tr.apply(wl.drift_exact(0.4), a); tr.apply(wl.drift_exact(0.6), a)
    tr.apply(wl.drift_exact(1.0), b)
    assert np.allclose(a, b, rtol=0, atol=1e-15)
    tr.apply(wl.drift_exact(-1.0), b)
    assert np.allclose(b, c, rtol=0, atol=1e-15)
    # the reference particle stays the reference particle
    z = np.zeros((6, 1))
    tr.apply(wl.drift_exact(5.0), z)
    assert np.all(z == 0.0)


# ------------------------------------------------------------------------------ R3x chromatic quad, R5x multipole (NEXT-3)
def fd_jacobian(el, c0, h=1e-6):
    J = np.zeros((6, 6))
    for j in range(6):
        cp, cm = np.array(c0, float).reshape(6, 1), np.array(c0, float).reshape(6, 1)
        cp[j] += h; cm[j] -= h
        oracle.Tracker(LAT).apply(el, cp)
        oracle.Tracker(LAT).apply(el, cm)
        J[:, j] = (cp[:, 0] - cm[:, 0]) / (2 * h)
    return J


@pytest.mark.parametrize("k", [1.2, -1.2, 0.0])
def test_chromatic_quad_on_momentum_is_r3_and_off_momentum_rescales_k(k):
    L = 0.4
    M = fd_jacobian(wl.quad_chromatic(L, k), np.zeros(6))
    assert np.allclose(M, jacobian([wl.quad(L, k)]), atol=1e-9)          # at pt = 0 it is the quadrupole of R3
    # off momentum: the transverse 4x4 is the R3 matrix of strength k/(1+delta) with px measured in units of p0(1+delta)
    pt = 0.05
    b0 = BG0 / math.sqrt(1 + BG0 ** 2)
    d1 = math.sqrt((1 / b0 - pt) ** 2 - 1 / BG0 ** 2)
    c0 = np.array([0, 0, 0, 0, 0, pt])
    J = fd_jacobian(wl.quad_chromatic(L, k), c0)
    Q = jacobian([wl.quad(L, k / d1)])
    S = np.diag([1, d1, 1, d1])                                          # (x, px) -> (x, px/(1+delta)) and back
    assert np.allclose(J[:4, :4], S @ Q[:4, :4] @ np.linalg.inv(S), atol=1e-8)


def test_chromatic_quad_is_symplectic_including_the_time_of_flight_term():
    """a wrong or missing betatron term in t breaks M^T S M = S through the (t, x..py) couplings"""
    c0 = np.array([2e-3, 1e-2, -1e-3, -2e-2, 3e-4, 4e-2])
    for k in (2.0, -2.0):
        J = fd_jacobian(wl.quad_chromatic(0.7, k), c0)
        assert np.max(np.abs(J.T @ S6 @ J - S6)) < 2e-8
        assert abs(J[4, 0]) > 1e-6 and abs(J[4, 3]) > 1e-6               # the couplings are really there


def test_chromatic_quad_zero_strength_on_axis_is_the_exact_drift():
    c = np.zeros((6, 5)); c[5] = [-0.1, -0.01, 0.0, 0.02, 0.2]
    a, b = c.copy(), c.copy()
    oracle.Tracker(LAT).apply(wl.quad_chromatic(1.3, 0.0), a)
    oracle.Tracker(LAT).apply(wl.drift_exact(1.3), b)
    assert np.allclose(a, b, rtol=0, atol=1e-15)                          # px = py = 0: pure time of flight


def test_multipole_kicks():
    c = rand_coords(16, 4, scale=np.array([1e-2, 1e-3, 1e-2, 1e-3, 1e-3, 1e-3]))
    x, y = c[0].copy(), c[2].copy()
    # quadrupole kick = thin limit of R3
    got = c.copy(); oracle.Tracker(LAT).apply(wl.multipole(2, 0.8), got)
    assert np.allclose(got[1], c[1] - 0.8 * x) and np.allclose(got[3], c[3] + 0.8 * y)
    L = 1e-7
    assert np.allclose(fd_jacobian(wl.multipole(2, 0.8), np.zeros(6)), jacobian([wl.quad(L, 0.8 / L)]), atol=2e-6)
    # sextupole: px -= kn (x^2 - y^2)/2, py += kn x y; skew quadrupole: px -= -ks y ... from the complex form
    got = c.copy(); oracle.Tracker(LAT).apply(wl.multipole(3, 5.0), got)
    assert np.allclose(got[1], c[1] - 5.0 * (x * x - y * y) / 2) and np.allclose(got[3], c[3] + 5.0 * x * y)
    got = c.copy(); oracle.Tracker(LAT).apply(wl.multipole(2, 0.0, 0.3), got)
    assert np.allclose(got[1], c[1] + 0.3 * y) and np.allclose(got[3], c[3] + 0.3 * x)
    # dipole kick is a constant; positions, t, pt never change; every kick is symplectic (derives from a potential)
    got = c.copy(); oracle.Tracker(LAT).apply(wl.multipole(1, 1e-3, 2e-3), got)
    assert np.allclose(got[1], c[1] - 1e-3) and np.allclose(got[3], c[3] + 2e-3)
    for el in (wl.multipole(3, 5.0, -2.0), wl.multipole(4, 40.0, 10.0)):
        J = fd_jacobian(el, [3e-3, 0, -2e-3, 0, 0, 0], h=1e-5)
        assert np.max(np.abs(J.T @ S6 @ J - S6)) < 1e-7
        got = c.copy(); oracle.Tracker(LAT).apply(el, got)
        assert np.array_equal(got[[0, 2, 4, 5]], c[[0, 2, 4, 5]])
