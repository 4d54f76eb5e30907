"""Pins of the CPU oracle against what the paper and the mathematics fix (-m "not gpu").

Each test cites the passage of PAPER.md it pins.  None of them retypes the oracle's own formula and compares it
with itself: they use quadrature, finite differences, brute force, conservation laws, closed-form solutions and
independently integrated ODEs.
"""
import math
import os

import numpy as np
import pytest
from scipy.integrate import solve_ivp

import oracle as O
from paper_2511_22852_b200 import workloads as W

from conftest import read_golden_table

C0, C2, C4 = W.EOS_C0, W.EOS_C2, W.EOS_C4


# ------------------------------------------------------------------------------------------------- kernel ----
@pytest.mark.parametrize("D", [1, 2, 3])
def test_kernel_normalisation(D):
    """Eq. 63 (:841): int W dV = 1, with Eq. 77 (:910) and sigma_d of :913."""
    h = 0.3
    r = np.linspace(0.0, 2.0 * h, 20001)
    Wv = np.array([O.kernel_W(D, h, x) for x in r])
    shell = {1: 2.0 * np.ones_like(r), 2: 2.0 * np.pi * r, 3: 4.0 * np.pi * r * r}[D]
    integral = np.trapezoid(Wv * shell, r)
    assert abs(integral - 1.0) < 2e-8
    assert O.kernel_W(D, h, 2.0 * h) == 0.0 and O.kernel_W(D, h, 2.5 * h) == 0.0


def test_kernel_sigma_d_golden(golden_dir):
    """W(0) = sigma_d (Eq. 77): values worked by hand in tests/golden/gubser_constants.txt."""
    g = {k: float(v) for k, v in read_golden_table(os.path.join(golden_dir, "gubser_constants.txt"))}
    assert abs(O.kernel_W(2, 0.3, 0.0) - g["sigma_2(h=0.3)"]) < 1e-8
    assert abs(O.kernel_W(3, 0.3, 0.0) - g["sigma_3(h=0.3)"]) < 1e-8


@pytest.mark.parametrize("D", [2, 3])
def test_kernel_gradient_matches_finite_difference(D):
    """Eq. 79 (:920) is the gradient of Eq. 77: central differences of W, both branches, C1 at q = 1, 2."""
    h = 0.3
    rng = np.random.default_rng(1)
    for _ in range(200):
        dr = np.zeros(3)
        dr[:D] = rng.normal(size=D)
        dr *= rng.uniform(0.02, 2.2) * h / np.linalg.norm(dr)
        g = O.kernel_gradW(D, h, dr)
        eps = 1e-6
        for i in range(D):
            dp, dm = dr.copy(), dr.copy()
            dp[i] += eps
            dm[i] -= eps
            fd = (O.kernel_W(D, h, np.linalg.norm(dp)) - O.kernel_W(D, h, np.linalg.norm(dm))) / (2 * eps)
            assert abs(g[i] - fd) < 2e-5 * O.kernel_W(D, h, 0.0) / h
        assert np.all(g[D:] == 0.0)
    for q in (1.0, 2.0):   # continuity of the gradient across the branch points
        a = O.kernel_gradW(D, h, [q * h * (1 - 1e-9), 0, 0])[0]
        b = O.kernel_gradW(D, h, [q * h * (1 + 1e-9), 0, 0])[0]
        assert abs(a - b) < 1e-6 * O.kernel_W(D, h, 0.0) / h
    assert np.all(O.kernel_gradW(D, h, [0, 0, 0]) == 0.0)


# --------------------------------------------------------------------------------------------- neighbours ----
def _oracle_for_cloud(pos, D, h=0.3, mode=0):
    p = W.base_params(dim=D, coords=0, eom=0, eos_kind=0, h=h, x0_start=0.0)
    p["neighbour_mode"] = mode
    o = O.Oracle(**p)
    f = {O.R1: pos[:, 0], O.R2: pos[:, 1], O.S: np.ones(len(pos))}
    if D == 3:
        f[O.R3] = pos[:, 2]
    o.load_particles(f)
    return o


@pytest.mark.parametrize("D", [2, 3])
def test_neighbour_cell_list_equals_brute_force(D):
    """:1434 (cell list, O(N)) against the O(N^2) definition Eq. 134 (:1224) with the strict r < 2h of reading 8."""
    rng = np.random.default_rng(7 + D)
    n = 3000 if D == 2 else 2500
    pos = rng.uniform(0.0, 6.0 if D == 2 else 2.4, size=(n, 3))
    a = _oracle_for_cloud(pos, D, mode=0).read_neighbors()
    b = _oracle_for_cloud(pos, D, mode=1).read_neighbors()
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1]) and np.array_equal(a[2], b[2])
    # and against numpy brute force in the same operation order
    d2 = (pos[:, None, 0] - pos[None, :, 0]) ** 2 + (pos[:, None, 1] - pos[None, :, 1]) ** 2
    if D == 3:
        d2 = d2 + (pos[:, None, 2] - pos[None, :, 2]) ** 2
    twoh = 2.0 * 0.3
    adj = d2 < twoh * twoh
    np.fill_diagonal(adj, False)
    assert np.array_equal(adj.sum(axis=1), a[0])
    ii, jj = np.nonzero(adj)
    assert np.array_equal(jj.astype(np.int32), a[2])


def test_neighbour_lattice_c1_and_counts():
    """Config 1's lattice has pairs at exactly r = 3 dx = 2h; both searches must take the same fp64 decision,
    and interior counts must be the lattice-point count (24 strictly inside, at most 28 with the r = 2h ring)."""
    w = W.config_c1()
    res = []
    for mode in (0, 1):
        p = dict(w.params)
        p["neighbour_mode"] = mode
        o = O.Oracle(**p)
        o.load_particles(w.fields)
        res.append(o.read_neighbors())
    for k in range(3):
        assert np.array_equal(res[0][k], res[1][k])
    x, y = w.fields[O.R1], w.fields[O.R2]
    interior = (np.abs(x) < 4.0) & (np.abs(y) < 4.0)
    cnt = res[0][0][interior]
    assert cnt.min() >= 24 and cnt.max() <= 28


def test_neighbour_count_exact_binary_lattice():
    """Lattice with dx = 1/8 (exact in binary) and h = 0.3: interior count = #{(i,j) != 0: i^2 + j^2 < (2h/dx)^2}."""
    dx, h = 0.125, 0.3
    n = 33
    x1 = (np.arange(n) - 16) * dx
    X, Y = np.meshgrid(x1, x1)
    pos = np.stack([X.ravel(), Y.ravel(), np.zeros(n * n)], axis=1)
    counts, _, _ = _oracle_for_cloud(pos, 2, h=h).read_neighbors()
    lim = (2 * h / dx) ** 2
    expect = sum(1 for i in range(-6, 7) for j in range(-6, 7) if (i or j) and i * i + j * j < lim)
    assert counts[(n * n) // 2] == expect == 68


def test_neighbour_estimate_table4(golden_dir):
    """Table 4 (:1251) / Eq. 136: cubic estimate (4h)^3/(dx^2 dz) = 1728 for h = 0.3, dx = dz = 0.1; the sphere
    estimate Eq. 133 (:1208) is 905; the oracle's interior count on that lattice must sit within 2 % of Eq. 133
    and below Eq. 136."""
    rows = read_golden_table(os.path.join(golden_dir, "table4_nnb_est.txt"))
    est, h, dx, dz = (float(v) for v in rows[0])
    assert abs((4 * h) ** 3 / (dx * dx * dz) - est) < 1e-9 * est
    for r in rows[1:]:
        e2, h2, dx2, dz2 = (float(v) for v in r)
        assert abs((4 * h2) ** 3 / (dx2 * dx2 * dz2) - e2) < 1e-9 * e2
    n = 15
    x1 = (np.arange(n) - 7) * dx
    X, Y, Z = np.meshgrid(x1, x1, x1, indexing="ij")
    pos = np.stack([X.ravel(), Y.ravel(), Z.ravel()], axis=1)
    counts, _, _ = _oracle_for_cloud(pos, 3, h=h).read_neighbors()
    centre = counts[(n ** 3) // 2]
    sphere = 4.0 / 3.0 * math.pi * (2 * h) ** 3 / (dx * dx * dz)
    assert abs(centre - sphere) < 0.02 * sphere and centre < est
    assert centre in (894, 900)   # 894 strictly inside; the six (+-6,0,0) points sit exactly on r = 2h


# ------------------------------------------------------------------------------------------ density sums ----
@pytest.mark.parametrize("D,dx,tol", [(2, 0.1, 2e-4), (2, 0.2, 5e-3), (3, 0.1, 2e-4)])
def test_partition_of_unity(D, dx, tol):
    """Eq. 72-76 (:882-904): sigma* = 1/V*, so sigma* dV -> 1 on a uniform lattice (m = 1)."""
    n = 21 if D == 2 else 15
    x1 = (np.arange(n) - (n - 1) / 2) * dx
    grids = np.meshgrid(*([x1] * D), indexing="ij")
    pos = np.zeros((grids[0].size, 3))
    for k in range(D):
        pos[:, k] = grids[k].ravel()
    o = _oracle_for_cloud(pos, D, h=0.3)
    sig = o.read_fields([O.SIGMA_STAR])[O.SIGMA_STAR]
    centre = np.argmin((pos ** 2).sum(axis=1))
    assert abs(sig[centre] * dx ** D - 1.0) < tol


def test_smoothed_entropy_integral():
    """Eq. 71 with Eq. 63: sum_a s*_a dV = sum_b S_b up to the partition-of-unity error, for a profile that is
    compact inside the lattice (so that no kernel mass leaks over the lattice edge)."""
    n, dx = 60, 0.1
    x1 = (np.arange(n) - 0.5 * (n - 1)) * dx
    X, Y = np.meshgrid(x1, x1)
    S = (np.exp(-(X ** 2 + Y ** 2) / (2 * 0.5 ** 2)) + 1e-7).ravel() * 50.0 * dx * dx
    p = W.base_params(dim=2, coords=0, eom=0, eos_kind=0)
    o = O.Oracle(**p)
    o.load_particles({O.R1: X.ravel(), O.R2: Y.ravel(), O.S: S})
    f = o.read_fields([O.S_STAR])
    assert abs((f[O.S_STAR] * dx * dx).sum() / S.sum() - 1.0) < 5e-4


# -------------------------------------------------------------------------------------------------- EoS ----
def _params():
    return O.make_params(**W.base_params())


def test_eos_closed_form_identities_and_round_trip():
    """App. A (:2115-2132): e = 3p, Gibbs-Duhem w = Ts + mu n, forward/inverse round trip <= 1e-13, and the
    conformal (Euler) identity dw/ds = 4T/3, dw/dn_q = 4 mu_q / 3 that the oracle obtains from the Hessian."""
    P = _params()
    rng = np.random.default_rng(3)
    for _ in range(300):
        T = rng.uniform(0.2, 3.0)
        mu = rng.uniform(-1.0, 1.0, size=3) * T
        p, s, nB, nS, nQ = O.eos_forward(P, T, mu)
        out = O.eos_closed_form(P, s, [nB, nS, nQ])
        assert abs(out[0] / T - 1) < 1e-13
        assert np.all(np.abs(out[1:4] - mu) < 1e-12 * T)
        assert abs(out[6] - 3 * out[4]) <= 1e-14 * out[6]
        assert abs(out[4] / p - 1) < 1e-12
        w = out[6] + out[4]
        assert abs(w - (out[0] * s + out[1] * nB + out[2] * nS + out[3] * nQ)) < 1e-12 * w
        assert abs(out[7] - 4 * T / 3) < 1e-11 * T
        assert np.all(np.abs(out[8:11] - 4 * mu / 3) < 1e-11 * T)
        assert out[5] == 1.0 / 3.0


def test_eos_forward_is_gradient_of_pressure():
    """Eq. A.6-A.7: s = dp/dT, n_q = dp/dmu_q (central differences of the forward pressure)."""
    P = _params()
    T, mu = 1.3, np.array([0.4, -0.2, 0.3])
    base = O.eos_forward(P, T, mu)
    e = 1e-6
    ds = (O.eos_forward(P, T + e, mu)[0] - O.eos_forward(P, T - e, mu)[0]) / (2 * e)
    assert abs(ds - base[1]) < 1e-7 * base[1]
    for q in range(3):
        mp, mm = mu.copy(), mu.copy()
        mp[q] += e
        mm[q] -= e
        dn = (O.eos_forward(P, T, mp)[0] - O.eos_forward(P, T, mm)[0]) / (2 * e)
        assert abs(dn - base[2 + q]) < 1e-7 * abs(base[1])


def test_eos_dw_ds_finite_difference():
    """dw/ds|_n and dw/dn_q|_s of the closed form against central differences of w(s, n)."""
    P = _params()
    s, n = 40.0, np.array([0.8, -0.3, 0.5])
    out = O.eos_closed_form(P, s, n)

    def w(ss, nn):
        o = O.eos_closed_form(P, ss, nn)
        return o[6] + o[4]
    e = 1e-5
    assert abs((w(s + e, n) - w(s - e, n)) / (2 * e) - out[7]) < 1e-7 * out[7]
    for q in range(3):
        npl, nm = n.copy(), n.copy()
        npl[q] += e
        nm[q] -= e
        assert abs((w(s, npl) - w(s, nm)) / (2 * e) - out[8 + q]) < 1e-6 * out[7]


def test_eos_golden_values(golden_dir):
    """s(T0) and e(T0) at T0 = 0.4 GeV, mu = 0 (hand-worked, tests/golden/gubser_constants.txt)."""
    g = {k: float(v) for k, v in read_golden_table(os.path.join(golden_dir, "gubser_constants.txt"))}
    p, s, *_ = O.eos_forward(_params(), g["T(1,0)"], [0, 0, 0])
    assert abs(s - g["s(T0)"]) < 1e-5 and abs(3 * p - g["e(T0)"]) < 1e-5
    out = O.eos_closed_form(_params(), g["s(T0)"], [0, 0, 0])
    assert abs(out[0] - g["T(1,0)"]) < 1e-8


def _small_table(ns=12, nq=5, with_wq=True):
    return W.make_eos_table(ns=ns, nq=nq, with_wq=with_wq)


def _table_oracle(tb, **kw):
    p = W.base_params(dim=2, coords=0, eom=0, eos_kind=1, **kw)
    o = O.Oracle(**p)
    o.load_eos_table(tb["axes"], tb["axis_kind"], tb["col_ids"], tb["data"])
    return o


def test_table_lookup_exact_at_nodes_and_multilinear():
    """:583-593: interpolation only.  Exact at nodes; exact for a function multilinear in the table coordinates."""
    tb = _small_table()
    o = _table_oracle(tb)
    ax = tb["axes"]
    rng = np.random.default_rng(5)
    for _ in range(50):
        # end nodes of the ratio axes are avoided: (y s)/s may round one ulp outside the table and be clamped
        idx = [rng.integers(0, len(ax[0]))] + [rng.integers(1, len(a) - 1) for a in ax[1:]]
        s = ax[0][idx[0]]
        n = [ax[k][idx[k]] * s for k in (1, 2, 3)]
        out, oob = o.eos_table_lookup(s, n)
        assert oob == 0
        assert np.allclose(out, tb["data"][idx[0], idx[1], idx[2], idx[3]], rtol=1e-13, atol=1e-300)
    # multilinear test function in (s, yB, yS, yQ)
    S_, YB, YS, YQ = np.meshgrid(*ax, indexing="ij")
    f = lambda s, a, b, c: 1.0 + 2.0 * s + 3.0 * a - b + 0.5 * c + s * a - 2 * a * b + s * a * b * c
    data = np.repeat(f(S_, YB, YS, YQ)[..., None], 8, axis=-1)
    o2 = _table_oracle(dict(tb, data=data, col_ids=list(range(8))))
    o2.load_eos_table(ax, tb["axis_kind"], list(range(8)), data)
    for _ in range(100):
        s = rng.uniform(ax[0][2], ax[0][-2])
        y = rng.uniform(-0.04, 0.04, size=3)
        out, oob = o2.eos_table_lookup(s, list(y * s))
        assert oob == 0 and abs(out[0] - f(s, *y)) < 1e-12 * abs(f(s, *y))


def test_table_lookup_converges_to_closed_form_and_clamps():
    """Refining the grid brings the table to the analytic EoS that generated it (App. A); out of range clamps."""
    P = _params()
    s, n = 37.3, np.array([0.31, -0.12, 0.2])
    exact = O.eos_closed_form(P, s, n)
    errs = []
    for ns, nq in ((100, 9), (100, 17)):
        tb = W.make_eos_table(ns=ns, nq=nq, with_wq=True)
        out, oob = _table_oracle(tb).eos_table_lookup(s, list(n))
        assert oob == 0
        errs.append(abs(out[1] / exact[1] - 1))
    assert errs[1] < errs[0] and errs[1] < 5e-3
    tb = _small_table()
    out, oob = _table_oracle(tb).eos_table_lookup(1e9, [0, 0, 0])
    assert oob == 1 and np.isfinite(out).all()
    out, oob = _table_oracle(tb).eos_table_lookup(1.0, [0.2, 0, 0])   # y_B = 0.2 > 0.05
    assert oob == 1


def test_table_generator_nodes_match_oracle_closed_form():
    """The input generator's offline inversion (workloads.make_eos_table) against the oracle's closed form."""
    tb = _small_table(ns=20, nq=5)
    P = _params()
    rng = np.random.default_rng(11)
    for _ in range(40):
        i = [rng.integers(0, len(a)) for a in tb["axes"]]
        s = tb["axes"][0][i[0]]
        n = [tb["axes"][k][i[k]] * s for k in (1, 2, 3)]
        ref = O.eos_closed_form(P, s, n)
        node = tb["data"][i[0], i[1], i[2], i[3]]
        assert np.allclose(node, ref, rtol=2e-11, atol=1e-14)


# ------------------------------------------------------------------------------- pair forces, ideal flow ----
def _random_viscous_state(D, n_side=12, coords=0, seed=0):
    rng = np.random.default_rng(seed)
    dx = 0.15
    x1 = (np.arange(n_side) - (n_side - 1) / 2) * dx
    grids = np.meshgrid(*([x1] * D), indexing="ij")
    N = grids[0].size
    f = {}
    for k in range(D):
        f[O.R1 + k] = grids[k].ravel() + rng.uniform(-0.02, 0.02, N)
        f[O.U1 + k] = rng.normal(0, 0.3, N)
    vol = dx ** D
    f[O.S] = rng.uniform(20, 60, N) * vol
    for q in range(3):
        f[O.NB + q] = rng.uniform(-0.5, 0.5, N) * vol
    f[O.BULK] = rng.normal(0, 0.5, N) * vol
    for c in (O.PI11, O.PI12, O.PI22, O.PI33) + ((O.PI13, O.PI23) if D == 3 else ()):
        f[c] = rng.normal(0, 0.5, N) * vol
    for q in range(3):
        for k in range(D):
            f[O.JB1 + 3 * q + k] = rng.normal(0, 0.02, N) * vol
    f[O.MASS] = rng.uniform(0.8, 1.2, N)
    return f


@pytest.mark.parametrize("D,coords", [(2, 0), (2, 1), (3, 1)])
def test_pair_forces_sum_to_zero(D, coords):
    """:944: the n = -1 derivative is pair antisymmetric, so sum_a m_a RHS_a = 0 for the momentum and charge
    equations to round-off — full viscous state, unequal masses."""
    f = _random_viscous_state(D, n_side=10 if D == 2 else 7, coords=coords, seed=D)
    p = W.viscous_params(D, 1, 0.01)
    p.update(coords=coords, eos_kind=0)
    o = O.Oracle(**p)
    o.load_particles(f)
    out = o.read_fields([O.FM1, O.FM2, O.FM3, O.FK_B, O.FK_S, O.FK_Q])
    m = f[O.MASS]
    for k in (O.FM1, O.FM2, O.FM3)[:D] + (O.FK_B, O.FK_S, O.FK_Q):
        scale = np.abs(m * out[k]).sum() + 1e-300
        assert abs((m * out[k]).sum()) < 1e-13 * scale


def test_uniform_interior_at_rest_has_zero_acceleration():
    """Lattice symmetry: uniform fluid at rest -> zero acceleration of interior particles (Cartesian)."""
    n, dx = 25, 0.1
    x1 = (np.arange(n) - 12) * dx
    X, Y = np.meshgrid(x1, x1)
    p = W.base_params(dim=2, coords=0, eom=0, eos_kind=0)
    o = O.Oracle(**p)
    o.load_particles({O.R1: X.ravel(), O.R2: Y.ravel(), O.S: np.full(n * n, 30.0 * dx * dx)})
    f = o.read_fields([O.RATE + O.U1, O.RATE + O.U2])
    c = (n * n) // 2
    edge_scale = np.abs(f[O.RATE + O.U1]).max()
    assert edge_scale > 1e-2
    assert abs(f[O.RATE + O.U1][c]) < 1e-12 * edge_scale and abs(f[O.RATE + O.U2][c]) < 1e-12 * edge_scale


@pytest.mark.parametrize("hyper", [False, True])
def test_ideal_flow_conserves_entropy_and_charges_exactly(hyper):
    """Eq. 105-106 (:1057-1059): dS/dx0 = dN_q/dx0 = 0 for every particle, bit-exactly, in ideal flow."""
    w = W.config_c2(n=24, dx=0.2, nsteps=2, table=None, ns=30, nq=5)
    p = dict(w.params)
    p.update(eos_kind=0, coords=1 if hyper else 0)
    o = O.Oracle(**p)
    o.load_particles(w.fields)
    f = o.read_fields([O.RATE + O.S, O.RATE + O.NB, O.RATE + O.NS, O.RATE + O.NQ])
    for v in f.values():
        assert np.all(v == 0.0)
    o.step(2)
    g = o.read_fields([O.S, O.NB])
    assert np.array_equal(g[O.S], w.fields[O.S]) and np.array_equal(g[O.NB], w.fields[O.NB])


def test_momentum_conserved_and_energy_drift_second_order_cartesian():
    """§5.6.5 (:1049-1063): Cartesian ideal fluid: total momentum to round-off; with equal-S particles the
    energy error is a time-integration error: halving dt shrinks the drift by >= 3.5x (RK2)."""
    n, dx = 20, 0.2
    x1 = (np.arange(n) - 9.5) * dx
    X, Y = np.meshgrid(x1, x1)
    drifts = []
    for dt, ns in ((0.08, 5), (0.04, 10), (0.02, 20)):
        p = W.base_params(dim=2, coords=0, eom=0, eos_kind=0, dx0=dt)
        o = O.Oracle(**p)
        o.load_particles({O.R1: X.ravel(), O.R2: Y.ravel(), O.S: np.full(n * n, 50.0 * dx * dx)})
        t0 = o.conserved_totals()
        o.step(ns)
        t1 = o.conserved_totals()
        assert abs(t1[2]) < 1e-10 * t0[1] and abs(t1[3]) < 1e-10 * t0[1]
        assert t1[5] == t0[5]
        drifts.append(abs(t1[1] / t0[1] - 1.0))
    assert drifts[0] / drifts[1] > 3.5 and drifts[1] / drifts[2] > 3.5
    assert drifts[2] < 1e-4


# --------------------------------------------------------------------------------------- analytic flows ----
def _gubser_errors(n, dx, h, dt, nsteps):
    w = W.config_c1(hyperbolic=True, n=n, dx=dx, nsteps=nsteps, dt=dt)
    w.params["h"] = h
    o = O.Oracle(**w.params)
    o.load_particles(w.fields)
    o.step(nsteps)
    f = o.read_fields([O.R1, O.R2, O.U1, O.U2, O.T])
    tau = w.params["x0_start"] + nsteps * dt
    r = np.hypot(f[O.R1], f[O.R2])
    m = r < 2.0
    Tan, uran = W.gubser_T(tau, r[m]), W.gubser_ur(tau, r[m])
    ur = np.hypot(f[O.U1], f[O.U2])[m]
    return np.abs(f[O.T][m] / Tan - 1).max(), np.abs(ur - uran).max()


def test_ideal_gubser_flow_hyperbolic():
    """Eq. 116-120 (:1137-1153): (2+1)D hyperbolic ideal flow converges to the closed-form Gubser solution."""
    eT1, eu1 = _gubser_errors(50, 0.2, 0.3, 0.05, 8)
    eT2, eu2 = _gubser_errors(100, 0.1, 0.2, 0.025, 16)
    assert eT1 < 0.015 and eu1 < 0.03
    assert eT2 < 0.006 and eu2 < 0.02
    assert eT2 < 0.6 * eT1


def test_gubser_generator_against_golden(golden_dir):
    g = {k: float(v) for k, v in read_golden_table(os.path.join(golden_dir, "gubser_constants.txt"))}
    for r in (0, 1, 2, 5):
        assert abs(W.gubser_T(1.0, float(r)) - g[f"T(1,{r})"]) < 2e-9
    assert abs(W.gubser_ur(1.0, 1.0) - g["ur(1,1)"]) < 1e-9 and abs(W.gubser_ur(1.0, 2.0) - g["ur(1,2)"]) < 1e-9


def _bjorken_run(flags, dt, nsteps, eom=1, integrator=2, dnmr=None):
    n, dx, h, tau0 = 36, 0.1, 0.3, 0.6
    x1 = (np.arange(n) - 0.5 * (n - 1)) * dx
    X, Y = np.meshgrid(x1, x1)
    x, y = X.ravel(), Y.ravel()
    T0 = 0.30 / W.HBARC
    p = W.base_params(dim=2, coords=1, eom=eom, flags=flags, eos_kind=0, h=h, x0_start=tau0, dx0=dt,
                      integrator=integrator, eta_over_s=0.2, zeta_max=0.1, tau_Pi_coeff=1.0)
    if dnmr is not None:
        p["dnmr_coeffs"] = dnmr
    o = O.Oracle(**p)
    o.load_particles({O.R1: x, O.R2: y, O.S: np.full(x.size, 4 * C0 * T0 ** 3 * tau0 * dx * dx)})
    ic = int(np.argmin(x * x + y * y))
    Tini = o.read_fields([O.T])[O.T][ic]
    o.step(nsteps)
    f = o.read_fields([O.T, O.BULK, O.PI33, O.PI11, O.PI22, O.PI12, O.SIGMA])
    tau1 = tau0 + nsteps * dt
    return p, ic, Tini, tau0, tau1, {k: v[ic] for k, v in f.items()}


def _bjorken_ode(p, flags, Tini, tau0, tau1):
    def rhs(tau, yv):
        e, phi, Pi = yv
        T = (e / (3 * C0)) ** 0.25
        s = 4 * C0 * T ** 3
        w = 4 * e / 3
        eta = p["eta_over_s"] * s
        tpi = max(p["tau_pi_coeff"] * eta / w, p["tau_floor"])
        zeta = p["zeta_max"] * p["zeta_width"] ** 2 / (p["zeta_width"] ** 2 + (T - p["zeta_T_peak"]) ** 2) * s
        tPi = p["tau_Pi_coeff"] * tpi
        sh = 1.0 if flags & 1 else 0.0
        bk = 1.0 if flags & 2 else 0.0
        return [-(e + e / 3 + bk * Pi - sh * phi) / tau,
                sh * (-phi / tpi + 4 * eta / (3 * tpi * tau) - 4 * phi / (3 * tau)),
                bk * (-(Pi + zeta / tau) / tPi - Pi / tau)]
    sol = solve_ivp(rhs, [tau0, tau1], [3 * C0 * Tini ** 4, 0.0, 0.0], rtol=1e-11, atol=1e-14)
    e1, phi1, Pi1 = sol.y[:, -1]
    return (e1 / (3 * C0)) ** 0.25, phi1, Pi1


@pytest.mark.parametrize("flags", [0, 1, 2, 3])
def test_bjorken_flow_ideal_shear_bulk(flags):
    """0+1D boost-invariant limit on a wide uniform slab (hyperbolic coordinates): the centre particle follows
    the textbook Bjorken ODEs — ideal (s tau = const), Israel-Stewart shear (Eq. 50 :678) with
    phi = -tau^2 pi^{eta eta}, and bulk (Eq. 49 :676).  Pins Gamma_g, the Christoffel terms of D pi, sigma^{mu nu},
    the entropy-production equation Eq. 96-98 and the relaxation equations."""
    p, ic, Tini, tau0, tau1, f = _bjorken_run(flags, 0.01, 30, eom=1 if flags else 0)
    T1, phi1, Pi1 = _bjorken_ode(p, flags, Tini, tau0, tau1)
    assert abs(f[O.T] / T1 - 1) < 5e-6
    sig = f[O.SIGMA]
    if flags & 1:
        phi = -tau1 ** 2 * f[O.PI33] * sig
        assert abs(phi / phi1 - 1) < 1e-3
        assert abs(f[O.PI11] * sig / (0.5 * phi1) - 1) < 1e-3 and abs(f[O.PI22] * sig / (0.5 * phi1) - 1) < 1e-3
        assert abs(f[O.PI12] * sig) < 1e-6 * phi1
    if flags & 2:
        assert abs(f[O.BULK] * sig / Pi1 - 1) < 1e-3


def test_rk_order_on_bjorken():
    """Step 6: observed order of RK2 (midpoint) and RK4 by step halving on the Bjorken shear+bulk solution."""
    errs = {}
    for integ, dts in ((2, (0.04, 0.02, 0.01)), (4, (0.08, 0.04))):
        for dt in dts:
            ns = int(round(0.32 / dt))
            p, ic, Tini, tau0, tau1, f = _bjorken_run(3, dt, ns, integrator=integ)
            T1, phi1, Pi1 = _bjorken_ode(p, 3, Tini, tau0, tau1)
            errs[(integ, dt)] = abs(-tau1 ** 2 * f[O.PI33] * f[O.SIGMA] - phi1)
    assert 3.0 < errs[(2, 0.04)] / errs[(2, 0.02)] < 5.5 and 3.0 < errs[(2, 0.02)] / errs[(2, 0.01)] < 5.5
    assert errs[(4, 0.04)] < 0.02 * errs[(2, 0.04)]
    assert errs[(4, 0.08)] / errs[(4, 0.04)] > 8.0


def test_dnmr_reduces_to_minimal_is():
    """DESIGN reading 11: with delta_PiPi = tau_Pi, delta_pipi = 4/3 tau_pi and the other second-order
    coefficients zero the DNMR branch is the minimal IS branch, bit for bit."""
    a = _bjorken_run(3, 0.02, 5, eom=1)[5]
    b = _bjorken_run(3, 0.02, 5, eom=2, dnmr=[1.0, 0.0, 4.0 / 3.0, 0.0, 0.0, 0.0, 0.0, 0.0])[5]
    for k in a:
        assert a[k] == b[k]
    c = _bjorken_run(3, 0.02, 5, eom=2, dnmr=list(W.DNMR_DEFAULT))[5]
    assert c[O.PI33] != a[O.PI33]


def _viscous_gubser_solution(etas, C, That0):
    def rhs(rho, y):
        lnT, pb = y
        tR = C * etas / math.exp(lnT)
        th = math.tanh(rho)
        return [(pb - 2.0) / 3.0 * th, 4.0 / (3 * C) * th - pb / tR - 4.0 / 3.0 * pb * pb * th]
    sp = solve_ivp(rhs, [0, 5], [math.log(That0), 0.0], rtol=1e-11, atol=1e-13, dense_output=True)
    sm = solve_ivp(rhs, [0, -12], [math.log(That0), 0.0], rtol=1e-11, atol=1e-13, dense_output=True)

    def sol(rho):
        rho = np.asarray(rho, dtype=np.float64)
        out = np.where(rho >= 0, sp.sol(np.clip(rho, 0, 5)), sm.sol(np.clip(rho, -12, 0)))
        return np.exp(out[0]), out[1]
    return sol


def test_viscous_gubser_shear():
    """Eq. 112a,c (:1117-1121) at mu = 0 integrated in rho (Eq. 118), with pi-bar = tau^2 pi^{eta eta} / w in the
    sign convention of the printed ODE (DESIGN reading 19) and
    pi^{mu nu} = -(pi-bar w / 2)(Delta^{mu nu} + z^mu z^nu) + pi-bar w z^mu z^nu: the oracle's shear sector in a
    non-trivial (2+1)D hyperbolic flow against the semi-analytic solution (cf. Fig. 7-8)."""
    q, etas, C = 1.0, 0.2, 5.0
    sol = _viscous_gubser_solution(etas, C, 1.2 * 2.027)

    def fields(tau, x, y):
        r = np.hypot(x, y)
        rho = np.arcsinh(-(1 - q * q * tau * tau + q * q * r * r) / (2 * q * tau))
        That, pb = sol(rho)
        T = That / tau
        ur = W.gubser_ur(tau, r, q)
        with np.errstate(invalid="ignore", divide="ignore"):
            ux = np.where(r > 0, ur * x / r, 0.0)
            uy = np.where(r > 0, ur * y / r, 0.0)
        return T, ux, uy, pb, 4 * C0 * T ** 4

    n, dx, h, dt, nsteps, tau0 = 60, 0.1, 0.2, 0.02, 15, 1.0
    x1 = (np.arange(n) - 0.5 * (n - 1)) * dx
    X, Y = np.meshgrid(x1, x1)
    x, y = X.ravel(), Y.ravel()
    T, ux, uy, pb, w = fields(tau0, x, y)
    gam = np.sqrt(1 + ux ** 2 + uy ** 2)
    sig = 1.0 / (dx * dx) / (gam * tau0)
    p = W.base_params(dim=2, coords=1, eom=1, flags=1, eos_kind=0, h=h, x0_start=tau0, dx0=dt, eta_over_s=etas,
                      tau_pi_coeff=C, tau_floor=0.0)
    o = O.Oracle(**p)
    o.load_particles({O.R1: x, O.R2: y, O.U1: ux, O.U2: uy, O.S: 4 * C0 * T ** 3 * gam * tau0 * dx * dx,
                      O.PI11: -pb * w / 2 * (1 + ux ** 2) / sig, O.PI12: -pb * w / 2 * ux * uy / sig,
                      O.PI22: -pb * w / 2 * (1 + uy ** 2) / sig, O.PI33: pb * w / tau0 ** 2 / sig})
    o.step(nsteps)
    tau1 = tau0 + nsteps * dt
    f = o.read_fields([O.R1, O.R2, O.U1, O.T, O.PI11, O.PI12, O.PI33, O.SIGMA])
    Ta, uxa, uya, pba, wa = fields(tau1, f[O.R1], f[O.R2])
    m = np.hypot(f[O.R1], f[O.R2]) < 1.8
    sg = f[O.SIGMA]
    assert np.abs(f[O.T][m] / Ta[m] - 1).max() < 0.01
    assert np.abs(f[O.U1][m] - uxa[m]).max() < 0.015
    pixy_a = -pba * wa / 2 * uxa * uya
    assert np.abs(f[O.PI12] * sg - pixy_a)[m].max() < 0.06 * np.abs(pixy_a[m]).max()
    pi33_a = pba * wa
    assert np.abs(f[O.PI33] * sg * tau1 ** 2 - pi33_a)[m].max() < 0.02 * np.abs(pi33_a[m]).max()
    pixx_a = -pba * wa / 2 * (1 + uxa ** 2)
    assert np.abs(f[O.PI11] * sg - pixx_a)[m].max() < 0.03 * np.abs(pixx_a[m]).max()


def test_shifted_gubser_3d_rates():
    """Eq. 113-125 (:1127-1171): (3+1)D hyperbolic ideal terms (u^eta, G_u, metric derivative).  The oracle's
    accelerations at tau0 on a lattice initialised with the shifted Gubser solution must match the analytic
    Lagrangian derivative du^i/dtau = (d_tau + v.grad) u^i of that solution (finite differences of the closed
    form); compared at interior particles within the SPH discretisation error."""
    tau0, dx, de, h = 1.0, 0.1, 0.1, 0.25
    nx, ne = 23, 17
    x1 = (np.arange(nx) - (nx - 1) / 2) * dx
    e1 = (np.arange(ne) - (ne - 1) / 2) * de
    X, Y, E = np.meshgrid(x1, x1, e1, indexing="ij")
    x, y, e = X.ravel(), Y.ravel(), E.ravel()
    T, ux, uy, ue = W.shifted_gubser(tau0, x, y, e)
    gam = np.sqrt(1 + ux ** 2 + uy ** 2 + tau0 ** 2 * ue ** 2)
    p = W.base_params(dim=3, coords=1, eom=0, eos_kind=0, h=h, x0_start=tau0, dx0=0.01)
    o = O.Oracle(**p)
    o.load_particles({O.R1: x, O.R2: y, O.R3: e, O.U1: ux, O.U2: uy, O.U3: ue,
                      O.S: 4 * C0 * T ** 3 * gam * tau0 * dx * dx * de})
    f = o.read_fields([O.RATE + O.U1, O.RATE + O.U2, O.RATE + O.U3])
    eps = 1e-5
    def U(t, xx, yy, ee):
        return np.array(W.shifted_gubser(t, xx, yy, ee)[1:])
    v = np.array([ux, uy, ue]) / gam
    lag = (U(tau0 + eps, x + eps * v[0], y + eps * v[1], e + eps * v[2]) -
           U(tau0 - eps, x - eps * v[0], y - eps * v[1], e - eps * v[2])) / (2 * eps)
    m = (np.abs(x) < 0.45) & (np.abs(y) < 0.45) & (np.abs(e) < 0.35) & (np.hypot(x, y) > 0.15)
    scale = np.abs(lag[0][m]).max()
    assert np.abs(f[O.RATE + O.U1][m] - lag[0][m]).max() < 0.05 * scale
    assert np.abs(f[O.RATE + O.U2][m] - lag[1][m]).max() < 0.05 * scale
    assert np.abs(f[O.RATE + O.U3][m] - lag[2][m]).max() < 0.08 * np.abs(lag[2][m]).max()


def test_diffusion_telegraph_and_charge_conservation():
    """Eq. 51 (:680) with reading 12 (Fick sign): a small baryon ripple on a static uniform background decays at
    the telegraph-equation rate  tau l^2 - l + D k^2 = 0, D = kappa / (dn/d alpha);  the pair sums conserve the
    total charge instantaneously to round-off, and its drift over a run is an O(dt^2) integration error."""
    dx, h, L, tauT, kBB = 0.05, 0.1, 1.6, 0.5, 0.3
    nx, ny = 64, 28
    x1 = (np.arange(nx) - 0.5 * (nx - 1)) * dx
    y1 = (np.arange(ny) - 0.5 * (ny - 1)) * dx
    X, Y = np.meshgrid(x1, y1)
    x, y = X.ravel(), Y.ravel()
    T0, k = 0.3 / W.HBARC, 2 * np.pi / L
    s0 = 4 * C0 * T0 ** 3
    kap = [0.0] * 9
    kap[0] = kBB
    drift = []
    for dt, ns in ((0.01, 20), (0.005, 40)):
        p = W.base_params(dim=2, coords=0, eom=1, flags=4, eos_kind=0, h=h, x0_start=0.0, dx0=dt,
                          kappa_over_T2=kap, tau_q_times_T=[tauT] * 3)
        o = O.Oracle(**p)
        o.load_particles({O.R1: x, O.R2: y, O.S: np.full(x.size, s0 * dx * dx),
                          O.NB: 1e-3 * s0 * np.cos(k * x) * dx * dx})
        m = (np.abs(x) < 0.5 * L) & (np.abs(y) < 0.25)

        def amp():
            f = o.read_fields([O.RHO_B, O.R1, O.T, O.FK_B])
            c = np.cos(k * f[O.R1][m])
            return (f[O.RHO_B][m] * c).sum() / (c * c).sum(), f[O.T][m].mean(), f[O.FK_B]
        a0, T, fk = amp()
        assert abs(fk.sum()) <= 1e-12 * np.abs(fk).sum()
        t0 = o.conserved_totals()
        o.step(ns)
        a1, _, fk = amp()
        assert abs(fk.sum()) <= 1e-12 * np.abs(fk).sum()
        t1 = o.conserved_totals()
        drift.append(abs(t1[6] - t0[6]))
    tau, D = tauT / T, kBB * T * T / (2 * C2 * T ** 3)
    disc = np.sqrt(complex(1 - 4 * tau * D * k * k))
    l1, l2 = (1 + disc) / (2 * tau), (1 - disc) / (2 * tau)
    t = 0.2
    exact = (-l2 / (l1 - l2) * np.exp(-l1 * t) + l1 / (l1 - l2) * np.exp(-l2 * t)).real
    assert abs((1 - a1 / a0) / (1 - exact) - 1) < 0.12       # SPH gradient at k h = 0.39 damps a little less
    assert a1 / a0 < 1.0
    assert drift[1] < 0.4 * drift[0] and drift[1] < 1e-6 * np.abs(1e-3 * s0 * np.cos(k * x) * dx * dx).sum()


def test_kappa_matrix_golden(golden_dir):
    rows = read_golden_table(os.path.join(golden_dir, "kappa_over_T2.txt"))
    flat = [float(v) for r in rows[:3] for v in r]
    assert flat == W.KAPPA_OVER_T2 and [float(v) for v in rows[3]] == W.TAU_Q_TIMES_T


def test_applicability_diagnostics_on_bjorken():
    """PAPER.md Eq. 58-61 (:797-805) on the boost-invariant slab at rest in hyperbolic coordinates, where
    everything is closed form: theta = 1/tau and sigma^{mu nu} sigma_{mu nu} = 2/(3 tau^2)
    (sigma^{xx} = sigma^{yy} = 1/(3 tau), sigma^{eta eta} = -2/(3 tau^3)), so Kn_pi = tau_pi sqrt(2/3) / tau and
    Kn_Pi = tau_Pi / tau; with u = (1,0,0,0), pi^{0 mu} = 0 and pi^{mu nu} pi_{mu nu} =
    sigma^2 (PI11^2 + PI22^2 + 2 PI12^2 + tau^4 PI33^2), Re_Pi^-1 = |BULK sigma| / p.  A dropped metric factor, a
    missing 1/3 Delta theta or a wrong relaxation time fails one of these."""
    n, dx, h, tau0 = 36, 0.1, 0.3, 0.7
    x1 = (np.arange(n) - 0.5 * (n - 1)) * dx
    X, Y = np.meshgrid(x1, x1)
    x, y = X.ravel(), Y.ravel()
    T0 = 0.30 / W.HBARC
    p = W.base_params(dim=2, coords=1, eom=1, flags=3, eos_kind=0, h=h, x0_start=tau0, dx0=0.01, eta_over_s=0.2,
                      zeta_max=0.1, tau_Pi_coeff=1.5)
    N = x.size
    pi11, pi22, pi12, pi33, bulk = 0.013, -0.004, 0.002, -0.009 / tau0 ** 2, -0.006
    o = O.Oracle(**p)
    o.load_particles({O.R1: x, O.R2: y, O.S: np.full(N, 4 * C0 * T0 ** 3 * tau0 * dx * dx),
                      O.PI11: np.full(N, pi11), O.PI22: np.full(N, pi22), O.PI12: np.full(N, pi12),
                      O.PI33: np.full(N, pi33), O.BULK: np.full(N, bulk)})
    ic = int(np.argmin(x * x + y * y))
    f = o.read_fields([O.KN_PI, O.RE_PI, O.KN_BULK, O.RE_BULK, O.THETA, O.SIGMA, O.P, O.T, O.S_DENS, O.E])
    T, s, e, pr, sig = (f[k][ic] for k in (O.T, O.S_DENS, O.E, O.P, O.SIGMA))
    eta = p["eta_over_s"] * s
    tau_pi = max(p["tau_pi_coeff"] * eta / (e + pr), p["tau_floor"])
    tau_Pi = p["tau_Pi_coeff"] * tau_pi
    assert abs(f[O.THETA][ic] * tau0 - 1) < 1e-6
    assert abs(f[O.KN_PI][ic] / (tau_pi * np.sqrt(2.0 / 3.0) / tau0) - 1) < 1e-6
    assert abs(f[O.KN_BULK][ic] / (tau_Pi / tau0) - 1) < 1e-6
    pipi = sig ** 2 * (pi11 ** 2 + pi22 ** 2 + 2 * pi12 ** 2 + tau0 ** 4 * pi33 ** 2)
    assert abs(f[O.RE_PI][ic] / (np.sqrt(pipi) / pr) - 1) < 1e-12
    assert abs(f[O.RE_BULK][ic] / (abs(bulk * sig) / pr) - 1) < 1e-12


def test_applicability_diagnostics_vanish_for_uniform_fluid_at_rest():
    """Cartesian, uniform, at rest, no dissipative fields: sigma^{mu nu} = 0, theta = 0, pi = Pi = 0 in the interior,
    so all four numbers vanish (to the SPH noise of the velocity gradient, which is exactly 0 for u = 0)."""
    n, dx = 30, 0.1
    x1 = (np.arange(n) - 0.5 * (n - 1)) * dx
    X, Y = np.meshgrid(x1, x1)
    x, y = X.ravel(), Y.ravel()
    p = W.base_params(dim=2, coords=0, eom=1, flags=3, eos_kind=0, h=0.3, x0_start=1.0, dx0=0.01, eta_over_s=0.2)
    o = O.Oracle(**p)
    o.load_particles({O.R1: x, O.R2: y, O.S: np.full(x.size, 4 * C0 * (0.3 / W.HBARC) ** 3 * dx * dx)})
    ic = int(np.argmin(x * x + y * y))
    f = o.read_fields([O.KN_PI, O.RE_PI, O.KN_BULK, O.RE_BULK])
    for k in (O.KN_PI, O.RE_PI, O.KN_BULK, O.RE_BULK):
        assert abs(f[k][ic]) < 1e-12


def test_freezeout_element_on_bjorken():
    """PAPER.md Eq. 145-148 (:1466-1482) where everything is closed form — the boost-invariant ideal slab at rest in
    hyperbolic coordinates: d_i eps = 0, d_tau eps = -(eps + p)/tau (so the surface is space-like, n_mu =
    (+1, 0, 0, 0): the outward normal of a cooling fluid points to later times), u.n = 1 and
    |d sigma| = m / sigma.  A wrong sign in Eq. 147, a missing D sigma = -sigma theta or a rate taken per unit of
    proper time fails this."""
    p, ic, Tini, tau0, tau1, _ = _bjorken_run(0, 0.01, 0, eom=0)
    n, dx = 36, 0.1
    x1 = (np.arange(n) - 0.5 * (n - 1)) * dx
    X, Y = np.meshgrid(x1, x1)
    o = O.Oracle(**p)
    T0 = 0.30 / W.HBARC
    o.load_particles({O.R1: X.ravel(), O.R2: Y.ravel(), O.S: np.full(X.size, 4 * C0 * T0 ** 3 * tau0 * dx * dx)})
    ids = [O.FO_DE0, O.FO_DE1, O.FO_DE2, O.FO_DE3, O.FO_N0, O.FO_N1, O.FO_N2, O.FO_N3, O.FO_DSIGMA, O.E, O.P, O.SIGMA]
    f = {k: v[ic] for k, v in o.read_fields(ids).items()}
    assert abs(f[O.FO_DE0] / (-(f[O.E] + f[O.P]) / tau0) - 1) < 1e-6
    assert abs(f[O.FO_DE1]) < 1e-9 * abs(f[O.FO_DE0]) and abs(f[O.FO_DE2]) < 1e-9 * abs(f[O.FO_DE0]) and f[O.FO_DE3] == 0.0
    assert abs(f[O.FO_N0] - 1.0) < 1e-12 and abs(f[O.FO_N1]) < 1e-9 and abs(f[O.FO_N2]) < 1e-9
    assert abs(f[O.FO_DSIGMA] * f[O.SIGMA] - 1.0) < 1e-12          # m = 1


def test_freezeout_normal_on_gubser():
    """Ideal Gubser flow (Eq. 116-120): eps = 3 c0 T(tau, r)^4 is analytic, so d_mu eps is too.  At r = 1.55 fm the
    SPH values converge to the analytic ones at second order in h (h = 0.3 -> 0.15 with dx = h/3: errors of ~9 % and
    ~2.5 % of d_tau eps and d_r eps, ratio > 3), the gradient is radial, the normal is unit (n.n = +-1), and
    |d sigma| = m / (sigma |u.n|) agrees with the analytic normal to the same accuracy."""
    errs = []
    for n, dx, h in ((80, 0.1, 0.3), (160, 0.05, 0.15)):
        w = W.config_c1(hyperbolic=True, n=n, dx=dx)
        p = dict(w.params)
        p["h"] = h
        o = O.Oracle(**p)
        o.load_particles(w.fields)
        x, y = w.fields[O.R1], w.fields[O.R2]
        r = np.hypot(x, y)
        ia = int(np.argmin(np.abs(x - 1.55) + np.abs(y - 0.05)))
        ids = [O.FO_DE0, O.FO_DE1, O.FO_DE2, O.FO_N0, O.FO_N1, O.FO_N2, O.FO_DSIGMA, O.SIGMA]
        f = {k: v[ia] for k, v in o.read_fields(ids).items()}
        tau, ra, eps_ = 1.0, r[ia], 1e-5
        e = lambda t, rr: 3 * C0 * W.gubser_T(t, rr) ** 4
        de_t = (e(tau + eps_, ra) - e(tau - eps_, ra)) / (2 * eps_)
        de_r = (e(tau, ra + eps_) - e(tau, ra - eps_)) / (2 * eps_)
        der = (f[O.FO_DE1] * x[ia] + f[O.FO_DE2] * y[ia]) / ra
        errs.append((abs(f[O.FO_DE0] / de_t - 1), abs(der / de_r - 1)))
        assert abs(f[O.FO_DE1] * y[ia] - f[O.FO_DE2] * x[ia]) < 1e-3 * abs(de_r) * ra          # radial
        nn = f[O.FO_N0] ** 2 - f[O.FO_N1] ** 2 - f[O.FO_N2] ** 2
        assert abs(abs(nn) - 1) < 1e-12
        norm = np.sqrt(abs(de_t ** 2 - de_r ** 2))
        n0, nr = -de_t / norm, -de_r / norm
        ur = W.gubser_ur(tau, ra)
        un = np.sqrt(1 + ur ** 2) * n0 + ur * nr
        assert abs(f[O.FO_DSIGMA] * f[O.SIGMA] * abs(un) - 1) < (0.25 if h > 0.2 else 0.07)
    assert errs[0][0] < 0.12 and errs[0][1] < 0.12 and errs[1][0] < 0.03 and errs[1][1] < 0.03
    assert errs[0][0] / errs[1][0] > 3.0 and errs[0][1] / errs[1][1] > 3.0


def _source_setup(D, coords, n, dx, tau0=1.3, dt=0.1):
    x1 = (np.arange(n) - 0.5 * (n - 1)) * dx
    grids = np.meshgrid(*([x1] * D), indexing="ij")
    p = W.base_params(dim=D, coords=coords, eom=0, eos_kind=0, h=0.3, x0_start=tau0, dx0=dt)
    o = O.Oracle(**p)
    f = {O.R1 + k: grids[k].ravel() for k in range(D)}
    f[O.S] = np.full(grids[0].size, 1.0)
    o.load_particles(f)
    return o, [g.ravel() for g in grids], tau0, dt


@pytest.mark.parametrize("D,coords", [(2, 0), (2, 1), (3, 1)])
def test_source_smearing_closed_forms(D, coords):
    """PAPER.md Eq. 35 (:521).  (1) One parton sitting on a particle: j^mu there = eta p^mu sigma_D(h_s) / (dx0 sqrt(-g))
    with sigma_2 = 10/(7 pi h^2), sigma_3 = 1/(pi h^3) (Eq. 77) and sqrt(-g) = tau or 1; at distance >= 2 h_s: 0.
    (2) Partition of unity on the lattice (h_s = 1.4 fm >> dx): sum_i j^mu_i dV = eta sum_k p^mu_k / (dx0 sqrt(-g)) over the
    partons inside the time window, to 2e-6 of sum |p|.  (3) The window is x0 - dx0 < t_k <= x0 exactly.  (4) Linear in p."""
    n, dx, hs, eta = (41, 0.2, 1.4, 0.62) if D == 2 else (21, 0.4, 1.4, 0.62)
    o, xs, tau0, dt = _source_setup(D, coords, n, dx)
    sqrtg = tau0 if coords == 1 else 1.0
    ic = int(np.argmin(sum(x * x for x in xs)))
    r0 = [xs[k][ic] for k in range(D)] + [0.0] * (3 - D)
    p1 = np.array([[2.0], [0.3], [-0.4], [0.1]])
    j = o.smear_sources(p1, np.array(r0)[:, None], [tau0], hs, eta)
    sig = 10.0 / (7.0 * np.pi * hs * hs) if D == 2 else 1.0 / (np.pi * hs ** 3)
    assert np.allclose(j[:, ic], eta * p1[:, 0] * sig / (dt * sqrtg), rtol=1e-13)
    dist = np.sqrt(sum((xs[k] - r0[k]) ** 2 for k in range(D)))
    assert np.all(j[:, dist >= 2 * hs] == 0.0) and np.all(j[0, dist < 2 * hs - 1e-9] > 0.0)
    # (2) + (3): five partons near the centre, two of them outside the time window
    rng = np.random.default_rng(35)
    rp = np.zeros((3, 5)); rp[:D] = rng.uniform(-0.6, 0.6, (D, 5))
    pp = rng.normal(0, 1, (4, 5)); pp[0] = np.abs(pp[0]) + 1
    tt = np.array([tau0, tau0 - 0.5 * dt, tau0 - dt + 1e-12, tau0 - dt, tau0 + 1e-12])     # last two: outside
    j = o.smear_sources(pp, rp, tt, hs, eta)
    tot = j.sum(axis=1) * dx ** D
    ref = eta * pp[:, :3].sum(axis=1) / (dt * sqrtg)
    assert np.max(np.abs(tot - ref)) <= 2e-6 * eta * np.abs(pp[:, :3]).sum() / (dt * sqrtg)
    # (4)
    j2 = o.smear_sources(2.5 * pp, rp, tt, hs, eta)
    assert np.max(np.abs(j2 - 2.5 * j)) <= 1e-13 * np.max(np.abs(j2))
