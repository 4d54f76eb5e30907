"""Pins of the source terms in the oracle's equations of motion (-m "not gpu"): PAPER.md Eq. 38 (:623),
Eq. 42-44 (:645-649), Eq. 96 (:1003), fed by the smearing of Eq. 35 (:521).  Closed forms of a uniform fluid, the
boost-invariant ODE with a source, and the balance of the conserved totals."""
import numpy as np
import pytest
from scipy.integrate import solve_ivp

import oracle as O
from paper_2511_22852_b200 import workloads as W

C0, C2 = W.EOS_C0, W.EOS_C2


def _uniform(D, n, dx, T0, tau0=1.0, hyper=False, u=None):
    x1 = (np.arange(n) - 0.5 * (n - 1)) * dx
    g = np.meshgrid(*([x1] * D), indexing="ij")
    f = {O.R1 + k: g[k].ravel() for k in range(D)}
    N = g[0].size
    gam = 1.0
    if u is not None:
        for k in range(D):
            f[O.U1 + k] = np.full(N, u[k])
        gam = np.sqrt(1.0 + sum(x * x for x in u))
    f[O.S] = np.full(N, 4 * C0 * T0 ** 3 * gam * (tau0 if hyper else 1.0) * dx ** D)
    return f, N


def test_uniform_fluid_at_rest_heats_and_is_pushed_exactly():
    """Eq. 42-44 for a uniform fluid at rest (Cartesian, theta = 0, no gradients): d eps/dt = I^0, w du^i/dt = I^i,
    dn_q/dt = I_q.  Rates of the centre particle at the loaded state, closed form; and with I^i = 0, I_q = 0 the energy
    density grows linearly, eps(t) = eps(0) + I^0 t (the midpoint rule is exact for a constant rate of eps... of s only
    to O(dt^2), so the comparison is at that level)."""
    n, dx, T0 = 21, 0.1, 0.3 / W.HBARC
    f, N = _uniform(2, n, dx, T0)
    p = W.base_params(dim=2, coords=0, eom=0, eos_kind=0, h=0.3, x0_start=0.0, dx0=0.01)
    o = O.Oracle(**p)
    o.load_particles(f)
    ic = N // 2
    r = o.read_fields([O.T, O.SIGMA, O.E, O.P])
    T, sig, w = r[O.T][ic], r[O.SIGMA][ic], r[O.E][ic] + r[O.P][ic]
    I = np.zeros((4, N))
    I[0], I[1], I[2] = 3.0, 0.7, -0.4
    Iq = np.zeros((3, N))
    Iq[0], Iq[2] = 0.05, -0.02
    o.set_sources(I, Iq)
    k = o.read_fields([O.RATE + O.S, O.RATE + O.U1, O.RATE + O.U2, O.RATE + O.NB, O.RATE + O.NS, O.RATE + O.NQ])
    assert abs(k[O.RATE + O.S][ic] * sig * T / 3.0 - 1) < 1e-12            # sigma T dS/dt = I^0 (mu = 0)
    assert abs(k[O.RATE + O.U1][ic] * w / 0.7 - 1) < 1e-12                 # w du^x/dt = I^x
    assert abs(k[O.RATE + O.U2][ic] * w / -0.4 - 1) < 1e-12
    assert abs(k[O.RATE + O.NB][ic] * sig / 0.05 - 1) < 1e-12 and abs(k[O.RATE + O.NQ][ic] * sig / -0.02 - 1) < 1e-12
    assert k[O.RATE + O.NS][ic] == 0.0
    I[1] = I[2] = 0.0
    o.set_sources(I, None)
    e0 = o.read_fields([O.E])[O.E][ic]
    o.step(10)
    e1 = o.read_fields([O.E])[O.E][ic]
    assert abs((e1 - e0) / (3.0 * 0.1) - 1) < 1e-5
    o.set_sources(None, None)                                              # cleared: nothing changes any more
    o.step(3)
    assert abs(o.read_fields([O.E])[O.E][ic] / e1 - 1) < 1e-12


def test_bjorken_with_energy_source():
    """Boost-invariant slab with a uniform I^tau: u_mu I^mu = I^tau and d eps/dtau = -(eps + p)/tau + I^tau (Eq. 42 with
    theta = 1/tau) — pins the sqrt(-g) and gamma factors of the source in the entropy equation, Eq. 96."""
    n, dx, tau0, dt, ns, Itau = 36, 0.1, 0.6, 0.01, 30, 8.0
    T0 = 0.3 / W.HBARC
    f, N = _uniform(2, n, dx, T0, tau0=tau0, hyper=True)
    p = W.base_params(dim=2, coords=1, eom=0, eos_kind=0, h=0.3, x0_start=tau0, dx0=dt)
    o = O.Oracle(**p)
    o.load_particles(f)
    ic = int(np.argmin(f[O.R1] ** 2 + f[O.R2] ** 2))
    e0 = o.read_fields([O.E])[O.E][ic]
    I = np.zeros((4, N))
    I[0] = Itau
    o.set_sources(I, None)
    o.step(ns)
    e1 = o.read_fields([O.E])[O.E][ic]
    tau1 = tau0 + ns * dt
    sol = solve_ivp(lambda t, e: [-(4.0 / 3.0) * e[0] / t + Itau], [tau0, tau1], [e0], rtol=1e-11, atol=1e-13)
    assert abs(e1 / sol.y[0, -1] - 1) < 2e-5
    nosrc = e0 * (tau0 / tau1) ** (4.0 / 3.0)
    assert abs(sol.y[0, -1] / nosrc - 1) > 0.02


def test_moving_fluid_energy_and_momentum_balance():
    """A uniform fluid moving with u^x = 0.5 under a uniform source I^mu = (I^0, I^x, 0): the momentum and charge
    equations are in conservative form, so the totals obey d P_i/dt = sum (m/sigma*) I_i and dN_q/dt = sum (m/sigma*) I_q
    to round-off per evaluation; the energy is not evolved, and d E/dt = sum (m/sigma*) I^0 holds to the integration
    error — which pins u_mu I^mu (not I^0) in Eq. 96 together with I_i in the momentum equation: T^{00} = w gamma^2 - p
    depends on both."""
    n, dx, T0 = 21, 0.1, 0.3 / W.HBARC
    f, N = _uniform(2, n, dx, T0, u=(0.5, 0.0))
    I = np.zeros((4, N))
    I[0], I[1] = 2.0, 1.2
    Iq = np.zeros((3, N))
    Iq[1] = 0.03
    res = []
    for dt in (0.004, 0.002):
        p = W.base_params(dim=2, coords=0, eom=0, eos_kind=0, h=0.3, x0_start=0.0, dx0=dt)
        o = O.Oracle(**p)
        o.load_particles(f)
        o.set_sources(I, Iq)
        vol = 1.0 / o.read_fields([O.SIGMA_STAR])[O.SIGMA_STAR]
        t0 = o.conserved_totals()
        o.step(1)
        t1 = o.conserved_totals()
        res.append(((t1[1] - t0[1]) / dt / np.sum(vol * I[0]) - 1, (t1[2] - t0[2]) / dt / np.sum(vol * -I[1]) - 1,
                    (t1[7] - t0[7]) / dt / np.sum(vol * Iq[1]) - 1))
    # edges of the finite block expand, which changes E slightly as well: compare at the 1e-3 level, and see it shrink
    assert abs(res[1][0]) < 2e-3 and abs(res[1][1]) < 2e-3 and abs(res[1][2]) < 1e-6
    # with I^0 in place of u_mu I^mu = gamma I^0 - gamma v I^x the energy rate would be off by tens of percent
    gam = np.sqrt(1.25)
    assert abs((gam * 2.0 - 0.5 * 1.2) / 2.0 - 1) > 0.1


@pytest.mark.parametrize("D,coords", [(2, 0), (3, 1)])
def test_smeared_partons_deposit_their_four_momentum(D, coords):
    """Eq. 35 -> Eq. 38: partons smeared onto the particles and fed back as I^mu change the totals over one step by
    eta_norm sum_k p^mu_k (partition of unity of the smearing kernel on the lattice, a few 1e-3 at dx / h_source = 0.1):
    momentum exactly by the conservative form, energy to the integration error."""
    n, dx = (41, 0.14) if D == 2 else (17, 0.3)
    T0, tau0, dt, hs, eta = 0.3 / W.HBARC, 1.3, 0.01, 1.0, 0.62
    f, N = _uniform(D, n, dx, T0, tau0=tau0, hyper=bool(coords))
    p = W.base_params(dim=D, coords=coords, eom=0, eos_kind=0, h=0.45 if D == 3 else 0.3, x0_start=tau0, dx0=dt)
    o = O.Oracle(**p)
    o.load_particles(f)
    rng = np.random.default_rng(8)
    npart = 40
    r = np.zeros((3, npart))
    r[:D] = rng.uniform(-0.4, 0.4, (D, npart))
    pm = rng.normal(0, 1.0, (4, npart))
    pm[0] = np.abs(pm[0]) + 2.0
    if D == 2:
        pm[3] = 0.0
    j = o.smear_sources(pm, r, np.full(npart, tau0), hs, eta)
    o.set_sources(j, None)
    t0 = o.conserved_totals()
    o.step(1)
    t1 = o.conserved_totals()
    # lower-index momentum P_i = g_ii P^i; in hyperbolic coordinates at eta ~ 0 the energy is E = sum tau T^{tau tau} cosh eta
    dE = (t1[1] + t1[10]) - (t0[1] + t0[10])
    if coords == 1:
        # the undisturbed slab loses energy to longitudinal work (2+1D: tracked in t[10]) or keeps it (3+1D): subtract the
        # same step without sources
        o2 = O.Oracle(**p)
        o2.load_particles(f)
        a0 = o2.conserved_totals()
        o2.step(1)
        a1 = o2.conserved_totals()
        dE -= (a1[1] + a1[10]) - (a0[1] + a0[10])
    assert abs(dE / (eta * pm[0].sum()) - 1) < 0.02
    for i in range(2):
        assert abs((t1[2 + i] - t0[2 + i]) / (-eta * pm[1 + i].sum()) - 1) < 0.01
