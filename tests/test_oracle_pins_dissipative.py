"""Pins of the oracle's dissipative sector beyond its minimal-IS limits, of the hyperbolic energy bookkeeping and of
the (div v) accumulator (-m "not gpu").  Round-1 review: these parts of oracle/ccake_oracle.cpp were reached by no
test, while BASELINE.json's configs 3-5 run on them.

None of the tests retypes the oracle's expression: they use independently integrated ODEs of the boost-invariant
limit (textbook DNMR Bjorken equations), Lorentz covariance (the same physical fluid described at rest and from a
moving frame), closed forms of a static fluid in hyperbolic coordinates, energy-momentum conservation, hand-evaluated
tensors on a rigidly rotating disc, and finite differences of the oracle's own density sums.
"""
import math

import numpy as np
import pytest
from scipy.integrate import solve_ivp

import oracle as O
from paper_2511_22852_b200 import workloads as W

C0, C2, C4 = W.EOS_C0, W.EOS_C2, W.EOS_C4

# second-order coefficients that are all different from their minimal-IS values and from each other, so that every
# term of Eq. 52 contributes at the percent level on the slab: delta_PiPi/tau_Pi, lambda_Pipi/tau_Pi,
# delta_pipi/tau_pi, tau_pipi/tau_pi, lambda_piPi, phi_omega
DNMR_TEST = [0.8, 0.5, 1.6, 1.1, 2.0, 0.0, 0.0, 0.0]


def _slab(D, n, dx, tau0, T0):
    x1 = (np.arange(n) - 0.5 * (n - 1)) * dx
    g = np.meshgrid(*([x1] * D), indexing="ij")
    f = {O.R1 + k: g[k].ravel() for k in range(D)}
    f[O.S] = np.full(g[0].size, 4 * C0 * T0 ** 3 * tau0 * dx ** D)
    return f


def _dnmr_bjorken_ode(p, Tini, tau0, tau1, phi0=0.0, Pi0=0.0):
    """Boost-invariant DNMR equations (Denicol et al., the limit of PAPER.md Eq. 52 :689-693 for u = (1,0,0,0) in
    (tau, x, y, eta_s)): with phi = -tau^2 pi^{eta eta}, theta = 1/tau, pi^{mn} sigma_{mn} = phi / tau,
        d e / d tau   = -(e + p + Pi - phi) / tau
        tau_pi dphi   = -phi + 4 eta / (3 tau) - (delta_pipi + tau_pipi / 3) phi / tau + (2/3) lambda_piPi Pi / tau
        tau_Pi dPi    = -Pi - zeta / tau - delta_PiPi Pi / tau + lambda_Pipi phi / tau                              """
    c = p["dnmr_coeffs"]

    def rhs(tau, yv):
        e, phi, Pi = yv
        T = (e / (3 * C0)) ** 0.25
        s = 4 * C0 * T ** 3
        w = 4 * e / 3
        eta = p["eta_over_s"] * s
        tpi = max(p["tau_pi_coeff"] * eta / w, p["tau_floor"])
        zeta = p["zeta_max"] * p["zeta_width"] ** 2 / (p["zeta_width"] ** 2 + (T - p["zeta_T_peak"]) ** 2) * s
        tPi = p["tau_Pi_coeff"] * tpi
        return [-(e + e / 3 + Pi - phi) / tau,
                (-phi + 4 * eta / (3 * tau) - (c[2] + c[3] / 3) * tpi * phi / tau + (2.0 / 3.0) * c[4] * Pi / tau) / tpi,
                (-Pi - zeta / tau - c[0] * tPi * Pi / tau + c[1] * tPi * phi / tau) / tPi]
    sol = solve_ivp(rhs, [tau0, tau1], [3 * C0 * Tini ** 4, phi0, Pi0], rtol=1e-11, atol=1e-14)
    e1, phi1, Pi1 = sol.y[:, -1]
    return (e1 / (3 * C0)) ** 0.25, phi1, Pi1


@pytest.mark.parametrize("D", [2, 3])
def test_dnmr_second_order_terms_on_bjorken(D):
    """PAPER.md Eq. 52 (:689-693), :711-712: delta_PiPi, lambda_Pipi, delta_pipi, tau_pipi and lambda_piPi each add a
    known term to the boost-invariant ODEs.  eom = 2 with five non-trivial coefficients on a wide uniform slab, in
    (2+1)D and in (3+1)D (uniform in eta_s as well), centre particle against the integrated ODE."""
    n, dx, h, tau0, dt, nsteps = (36, 0.1, 0.3, 0.6, 0.01, 30) if D == 2 else (17, 0.15, 0.3, 0.6, 0.01, 20)
    T0 = 0.30 / W.HBARC
    p = W.base_params(dim=D, coords=1, eom=2, flags=3, eos_kind=0, h=h, x0_start=tau0, dx0=dt, eta_over_s=0.2,
                      zeta_max=0.5, tau_Pi_coeff=1.0, dnmr_coeffs=list(DNMR_TEST))
    f = _slab(D, n, dx, tau0, T0)
    o = O.Oracle(**p)
    o.load_particles(f)
    ic = int(np.argmin(sum(f[O.R1 + k] ** 2 for k in range(D))))
    Tini = o.read_fields([O.T])[O.T][ic]
    o.step(nsteps)
    tau1 = tau0 + nsteps * dt
    g = {k: v[ic] for k, v in o.read_fields([O.T, O.BULK, O.PI33, O.PI11, O.PI22, O.PI12, O.SIGMA]).items()}
    T1, phi1, Pi1 = _dnmr_bjorken_ode(p, Tini, tau0, tau1)
    sig = g[O.SIGMA]
    assert abs(g[O.T] / T1 - 1) < 1e-5
    assert abs(-tau1 ** 2 * g[O.PI33] * sig / phi1 - 1) < 1e-3
    assert abs(g[O.PI11] * sig / (0.5 * phi1) - 1) < 1e-3 and abs(g[O.PI22] * sig / (0.5 * phi1) - 1) < 1e-3
    assert abs(g[O.BULK] * sig / Pi1 - 1) < 1e-3
    # each coefficient matters at a level the tolerances resolve: switching any of them back to its minimal-IS value
    # moves the ODE solution by more than 5e-3 in phi or Pi
    for k, v in ((0, 1.0), (1, 0.0), (2, 4.0 / 3.0), (3, 0.0), (4, 0.0)):
        q = dict(p)
        q["dnmr_coeffs"] = list(DNMR_TEST)
        q["dnmr_coeffs"][k] = v
        _, phi_k, Pi_k = _dnmr_bjorken_ode(q, Tini, tau0, tau1)
        assert max(abs(phi_k / phi1 - 1), abs(Pi_k / Pi1 - 1)) > 5e-3, k


def test_dnmr_vorticity_term_on_rotating_disc():
    """The vorticity term of Eq. 52's G^{mu nu}, 2 tau_pi phi_omega pi^{<mu}_lambda omega^{nu> lambda} (DESIGN reading
    11), on a rigidly rotating uniform disc in Cartesian (2+1)D: at the centre u^i = 0, sigma^{ij} = 0, theta = 0 and
    omega^{xy} = 1/2 (grad^x u^y - grad^y u^x) = -Omega (mostly-minus metric, grad^i = -d_i), so with a uniform
    pi^{xx} = a, pi^{yy} = b, pi^{xy} = c the term evaluates by hand to
        Y^{xx} = pi^x_y omega^{xy} = c Omega,   Y^{yy} = -c Omega,   Y^{xy} = (b - a) Omega / 2,
    and d pi~^{ij}/dt (phi_omega = 1) - d pi~^{ij}/dt (phi_omega = 0) = 2 Y^{ij} / sigma.  The SPH velocity gradient of
    a linear field on this lattice is exact to 2e-3."""
    n, dx, h, Om = 41, 0.1, 0.3, 0.05
    x1 = (np.arange(n) - 0.5 * (n - 1)) * dx
    X, Y = np.meshgrid(x1, x1, indexing="ij")
    x, y = X.ravel(), Y.ravel()
    T0 = 0.30 / W.HBARC
    ux, uy = -Om * y, Om * x
    gam = np.sqrt(1 + ux ** 2 + uy ** 2)
    sig = 1.0 / (dx * dx) / gam
    a, b, c = 0.7, -0.4, 0.3
    base = {O.R1: x, O.R2: y, O.U1: ux, O.U2: uy, O.S: 4 * C0 * T0 ** 3 * gam * dx * dx,
            O.PI11: a / sig, O.PI22: b / sig, O.PI12: c / sig, O.PI33: -(a + b) / sig}
    ic = int(np.argmin(x * x + y * y))
    rates = {}
    for phi_om in (0.0, 1.0):
        coeffs = [1.0, 0.0, 4.0 / 3.0, 0.0, 0.0, phi_om, 0.0, 0.0]
        p = W.base_params(dim=2, coords=0, eom=2, flags=1, eos_kind=0, h=h, x0_start=0.0, dx0=0.01, eta_over_s=0.2,
                          dnmr_coeffs=coeffs)
        o = O.Oracle(**p)
        o.load_particles(base)
        rates[phi_om] = {k: v[ic] for k, v in o.read_fields([O.RATE + O.PI11, O.RATE + O.PI22, O.RATE + O.PI12,
                                                              O.SIGMA]).items()}
    s0 = rates[1.0][O.SIGMA]
    d = {k: (rates[1.0][k] - rates[0.0][k]) * s0 for k in (O.RATE + O.PI11, O.RATE + O.PI22, O.RATE + O.PI12)}
    assert abs(d[O.RATE + O.PI11] / (2 * c * Om) - 1) < 5e-3
    assert abs(d[O.RATE + O.PI22] / (-2 * c * Om) - 1) < 5e-3
    assert abs(d[O.RATE + O.PI12] / ((b - a) * Om) - 1) < 5e-3


def test_dnmr_tensor_terms_on_linear_flow():
    """Index structure of the second-order shear terms of Eq. 52 where nothing is diagonal: a uniform fluid with the
    linear velocity field u^i = L^i_j x^j (Cartesian (2+1)D, |L| << 1) and a uniform, non-diagonal pi^{ij}.  At the
    centre u = (1, 0, 0, 0), Du = 0 (uniform thermodynamics), so with the definitions of the Notation section (:164-169)
        grad^i u^j = -L^j_i,  theta = tr L,  sigma^{ij} = -(L + L^T)^{ij}/2 + delta^{ij} theta/3
    are plain 4x4 numpy arrays here, and each coefficient c of the shear equation changes sigma tau_pi d pi~^{ij}/dt by
    its own term: -tau_pipi pi^{l<i} sigma^{j>}_l, lambda_piPi Pi sigma^{ij}, -delta_pipi pi^{ij} theta."""
    n, dx, h = 41, 0.1, 0.3
    x1 = (np.arange(n) - 0.5 * (n - 1)) * dx
    X, Y = np.meshgrid(x1, x1, indexing="ij")
    x, y = X.ravel(), Y.ravel()
    T0 = 0.30 / W.HBARC
    L = np.array([[0.03, 0.05], [-0.02, 0.04]])              # L[i][j] = d_j u^i
    ux, uy = L[0, 0] * x + L[0, 1] * y, L[1, 0] * x + L[1, 1] * y
    gam = np.sqrt(1 + ux ** 2 + uy ** 2)
    sig = 1.0 / (dx * dx) / gam
    a, b, c, Pi0 = 0.7, -0.4, 0.3, 0.25
    base = {O.R1: x, O.R2: y, O.U1: ux, O.U2: uy, O.S: 4 * C0 * T0 ** 3 * gam * dx * dx, O.BULK: Pi0 / sig,
            O.PI11: a / sig, O.PI22: b / sig, O.PI12: c / sig, O.PI33: -(a + b) / sig}
    ic = int(np.argmin(x * x + y * y))

    def rates(coeffs):
        p = W.base_params(dim=2, coords=0, eom=2, flags=3, eos_kind=0, h=h, x0_start=0.0, dx0=0.01, eta_over_s=0.2,
                          zeta_max=0.1, dnmr_coeffs=coeffs)
        o = O.Oracle(**p)
        o.load_particles(base)
        r = o.read_fields([O.RATE + O.PI11, O.RATE + O.PI22, O.RATE + O.PI12, O.RATE + O.PI33, O.SIGMA, O.T, O.S_DENS, O.E, O.P])
        return {k: v[ic] for k, v in r.items()}

    ref = [1.0, 0.0, 4.0 / 3.0, 0.0, 0.0, 0.0, 0.0, 0.0]
    r0 = rates(ref)
    s0 = r0[O.SIGMA]
    tau_pi = max(5.0 * 0.2 * r0[O.S_DENS] / (r0[O.E] + r0[O.P]), 0.005)
    # tensors at the centre, index order (t, x, y, z), mostly-minus metric
    g = np.diag([1.0, -1.0, -1.0, -1.0])
    u = np.array([1.0, 0.0, 0.0, 0.0])
    du = np.zeros((4, 4))                      # du[m][n] = d_m u^n
    du[1:3, 1:3] = L.T
    gradu = g @ du                             # grad^m u^n = g^{mm} d_m u^n
    theta = np.trace(du)
    Delta = g - np.outer(u, u)
    sg = 0.5 * (gradu + gradu.T) - Delta * theta / 3.0
    pi = np.zeros((4, 4))
    pi[1, 1], pi[2, 2], pi[1, 2], pi[2, 1], pi[3, 3] = a, b, c, c, -(a + b)
    sg_lo = g @ sg                             # sigma_l^j  (first index lowered)
    Xf = pi.T @ sg_lo                          # X^{ij} = pi^{l i} sigma_l^j
    Xs = 0.5 * (Xf + Xf.T) - Delta / 3.0 * np.einsum("ab,ab->", pi, g @ sg @ g)
    comp = {O.RATE + O.PI11: (1, 1), O.RATE + O.PI22: (2, 2), O.RATE + O.PI12: (1, 2), O.RATE + O.PI33: (3, 3)}

    def check(coeffs, term, what):
        r1 = rates(coeffs)
        for k, (i, j) in comp.items():
            got = (r1[k] - r0[k]) * s0 * tau_pi               # sigma tau_pi gamma d pi~/dt at gamma = 1
            assert abs(got - term[i, j]) < 4e-3 * np.abs(term).max(), (what, k, got, term[i, j])

    c3 = list(ref); c3[3] = 1.3
    check(c3, -1.3 * tau_pi * Xs, "tau_pipi")
    c4 = list(ref); c4[4] = 0.9
    check(c4, 0.9 * Pi0 * sg, "lambda_piPi")
    c2 = list(ref); c2[2] = 4.0 / 3.0 + 0.5
    check(c2, -0.5 * tau_pi * pi * theta, "delta_pipi")


# ------------------------------------------------------------------------------ diffusion in a moving frame ----
def test_diffusion_christoffel_term_on_bjorken():
    """Eq. 51 (:680) on the boost-invariant slab in (3+1)D with a uniform J~^eta: u = (1,0,0,0), alpha uniform, so
    only the relaxation and the Christoffel term of D J~^eta = dJ~^eta/dtau + Gamma^eta_{tau eta} J~^eta act:
        dJ~^eta/dtau = -J~^eta / tau - J~^eta / tau_q,   tau_q = c / T(tau),   T = T0 (tau0/tau)^(1/3) (ideal Bjorken)
    => J~^eta(tau) = J~^eta_0 (tau0/tau) exp[-(3 T0 tau0^(1/3) / 2c)(tau^(2/3) - tau0^(2/3))], and J~^x decays without
    the 1/tau factor."""
    n, dx, h, tau0, dt, nsteps, cq = 21, 0.15, 0.3, 0.6, 0.005, 24, 0.5
    T0 = 0.30 / W.HBARC
    f = _slab(3, n, dx, tau0, T0)
    N = f[O.S].size
    J0 = 1e-3 * f[O.S][0]
    f[O.JB1 + 2] = np.full(N, J0)            # J~^eta_B
    f[O.JB1 + 3] = np.full(N, 0.5 * J0)      # J~^x_S
    kap = [0.0] * 9
    kap[0] = 0.3
    p = W.base_params(dim=3, coords=1, eom=1, flags=4, eos_kind=0, h=h, x0_start=tau0, dx0=dt, kappa_over_T2=kap,
                      tau_q_times_T=[cq] * 3)
    o = O.Oracle(**p)
    o.load_particles(f)
    ic = int(np.argmin(f[O.R1] ** 2 + f[O.R2] ** 2 + f[O.R3] ** 2))
    Tini = o.read_fields([O.T])[O.T][ic]
    o.step(nsteps)
    tau1 = tau0 + nsteps * dt
    g = o.read_fields([O.JB1 + 2, O.JB1 + 3, O.T])
    relax = math.exp(-(3 * Tini * tau0 ** (1 / 3) / (2 * cq)) * (tau1 ** (2 / 3) - tau0 ** (2 / 3)))
    assert abs(g[O.T][ic] / (Tini * (tau0 / tau1) ** (1 / 3)) - 1) < 1e-4
    assert abs(g[O.JB1 + 2][ic] / (J0 * (tau0 / tau1) * relax) - 1) < 3e-4
    assert abs(g[O.JB1 + 3][ic] / (0.5 * J0 * relax) - 1) < 3e-4


def _transverse_gradient_fluid(v, Jx_rest, Jy_rest, nx=24, ny=56, dx0=0.1):
    """A fluid that is static in its rest frame with a temperature gradient along y and a uniform diffusion current
    (J'^x, J'^y), described from a frame moving along x: Lorentz contraction of the lattice in x, u^x = gamma v,
    J^x = gamma J'^x, J^y = J'^y (J^0 follows from orthogonality).  Nothing depends on x, so equal lab times are equal
    rest-frame times."""
    gam = 1.0 / math.sqrt(1.0 - v * v)
    dx, dy = dx0 / gam, dx0
    x1 = (np.arange(nx) - 0.5 * (nx - 1)) * dx
    y1 = (np.arange(ny) - 0.5 * (ny - 1)) * dy
    X, Y = np.meshgrid(x1, y1, indexing="ij")
    x, y = X.ravel(), Y.ravel()
    T = (0.30 / W.HBARC) * (1.0 + 0.25 * np.tanh(y / 0.8))
    s = 4 * C0 * T ** 3
    sig = 1.0 / (dx0 * dy)                      # rest-frame reference density: one particle per rest-frame cell
    f = {O.R1: x, O.R2: y, O.U1: np.full(x.size, gam * v), O.U2: np.zeros(x.size), O.S: s / sig,
         O.JB1: np.full(x.size, gam * Jx_rest / sig), O.JB1 + 1: np.full(x.size, Jy_rest / sig)}
    return f, gam, sig


def test_moving_frame_diffusion_and_momentum_by_lorentz_covariance():
    """Moving-frame part of Eq. 51 (:680): D J~^i + u^i J~^nu Du_nu with J^0 from orthogonality, and the ideal
    momentum equation at u != 0.  The alpha-gradient vanishes (mu = 0), so reading 12's dropped d_0 alpha term plays
    no role and the equations are Lorentz covariant: in the rest frame (u' = 0, acceleration a'^y from the pressure
    gradient) D J~'^i = -J~'^i / tau_q and D J~'^0 = J~'^y a'^y; boosting with velocity v along x,
        du^y/dt  = a'^y / gamma,                du^x/dt = 0,
        dJ~^y/dt = -J~'^y / (gamma tau_q),      dJ~^x/dt = -J~'^x / tau_q + v J~'^y a'^y,   J~'^x = J~^x / gamma.
    The last term is the u^i J.Du term: it is 40 % of dJ~^x/dt here.  a'^y comes from a second run of the same fluid at
    rest (its own lattice), so the boosted momentum equation is pinned as well."""
    v, Jx, Jy, cq = 0.6, 0.02, 0.05, 2.0
    kap = [0.0] * 9
    kap[0] = 0.3
    p = W.base_params(dim=2, coords=0, eom=1, flags=4, eos_kind=0, h=0.3, x0_start=0.0, dx0=0.01, kappa_over_T2=kap,
                      tau_q_times_T=[cq] * 3)
    ids = [O.RATE + O.U1, O.RATE + O.U2, O.RATE + O.JB1, O.RATE + O.JB1 + 1, O.T, O.SIGMA, O.R1, O.R2]
    f0, _, sig0 = _transverse_gradient_fluid(0.0, Jx, Jy)
    o0 = O.Oracle(**p)
    o0.load_particles(f0)
    r0 = o0.read_fields(ids)
    f1, gam, _ = _transverse_gradient_fluid(v, Jx, Jy)
    o1 = O.Oracle(**p)
    o1.load_particles(f1)
    r1 = o1.read_fields(ids)
    m = (np.abs(f0[O.R2]) < 1.2) & (np.abs(f0[O.R1]) < 0.35)        # interior, same (i, j) on both lattices
    ay = r0[O.RATE + O.U2]                                            # rest-frame acceleration a'^y
    tq = cq / r0[O.T]
    assert np.abs(ay[m]).max() > 0.05
    # rest frame: plain relaxation
    assert np.allclose(r0[O.RATE + O.JB1][m], -(Jx / sig0) / tq[m], rtol=1e-9)
    assert np.allclose(r0[O.RATE + O.JB1 + 1][m], -(Jy / sig0) / tq[m], rtol=1e-9)
    # same thermodynamics on both lattices (rest-frame densities agree)
    assert np.allclose(r1[O.T][m], r0[O.T][m], rtol=2e-4) and np.allclose(r1[O.SIGMA][m], sig0, rtol=2e-3)
    scale = np.abs(ay[m]).max()
    assert np.abs(r1[O.RATE + O.U2][m] - ay[m] / gam).max() < 0.01 * scale
    assert np.abs(r1[O.RATE + O.U1][m]).max() < 0.01 * scale
    sig1 = r1[O.SIGMA]
    exp_y = -(Jy / sig1) / (gam * tq)
    exp_x = -(Jx / sig1) / tq + v * (Jy / sig1) * ay
    assert np.abs(r1[O.RATE + O.JB1 + 1][m] - exp_y[m]).max() < 0.01 * np.abs(exp_y[m]).max()
    assert np.abs(r1[O.RATE + O.JB1][m] - exp_x[m]).max() < 0.01 * np.abs(exp_x[m]).max()
    assert np.abs(v * (Jy / sig1) * ay)[m].max() > 0.3 * np.abs(exp_x[m]).max()     # the term under test matters


def test_boosted_telegraph_dispersion():
    """Eq. 51 (:680) with reading 12 in a uniformly moving fluid (u^x = gamma v), small baryon ripple, mu ~ 0.  Normal
    modes exp(w t + i k x) of the equations as read — charge conservation d_t (gamma n + v J) + d_x (gamma v n + J) = 0
    with J^0 = v J^x, and tau gamma (d_t + v d_x) J + J = -D gamma^2 d_x n (spatial projector -(1 + u_x^2) d_x alpha;
    the d_0 alpha part is dropped) — obey
        tau gamma^2 (w + i k v)^2 + gamma (w + i k v) - i D gamma^2 k v w + D gamma^2 k^2 = 0.
    The rest-frame density amplitude a(t) = c1 e^{w1 t} + c2 e^{w2 t} (c1 + c2 = A, J(0) = 0) is compared with the
    complex Fourier amplitude of the oracle's n_B: decay and phase of the ripple (SPH gradient error at k h = 0.39: a
    few percent, as in the static telegraph pin)."""
    dx, h, L, tauT, kBB, v = 0.05, 0.1, 1.6, 0.5, 0.3, 0.5
    gam = 1.0 / math.sqrt(1 - v * v)
    nx, ny = 72, 24
    x1 = (np.arange(nx) - 0.5 * (nx - 1)) * dx
    y1 = (np.arange(ny) - 0.5 * (ny - 1)) * dx
    X, Y = np.meshgrid(x1, y1)
    x, y = X.ravel(), Y.ravel()
    T0, k = 0.3 / W.HBARC, 2 * np.pi / L
    s0 = 4 * C0 * T0 ** 3
    kap = [0.0] * 9
    kap[0] = kBB
    dt, ns = 0.005, 40
    p = W.base_params(dim=2, coords=0, eom=1, flags=4, eos_kind=0, h=h, x0_start=0.0, dx0=dt, kappa_over_T2=kap,
                      tau_q_times_T=[tauT] * 3)
    o = O.Oracle(**p)
    # lab-frame lattice: one particle per lab cell dx^2, rest-frame densities s0 and n(x) -> per-particle S = s gamma dx^2
    o.load_particles({O.R1: x, O.R2: y, O.U1: np.full(x.size, gam * v), O.S: np.full(x.size, s0 * gam * dx * dx),
                      O.NB: 1e-3 * s0 * np.cos(k * x) * gam * dx * dx})

    def amp():
        f = o.read_fields([O.RHO_B, O.R1, O.R2, O.T])
        m = (np.abs(f[O.R1] - f[O.R1].mean()) < 0.5 * L) & (np.abs(f[O.R2]) < 0.2)
        e = np.exp(-1j * k * f[O.R1][m])
        return 2.0 * (f[O.RHO_B][m] * e).mean(), f[O.T][m].mean()
    a0, T = amp()
    o.step(ns)
    a1, _ = amp()
    t = ns * dt
    tau, D = tauT / T, kBB * T * T / (2 * C2 * T ** 3)
    # quadratic A w^2 + B w + C = 0 of the dispersion relation above
    A = tau * gam ** 2
    B = 2j * tau * gam ** 2 * k * v + gam - 1j * D * gam ** 2 * k * v
    Cc = -tau * gam ** 2 * k * k * v * v + 1j * gam * k * v + D * gam ** 2 * k * k
    w1, w2 = np.roots([A, B, Cc])
    g1, g2 = 1.0 / (tau * gam * (w1 + 1j * k * v) + 1), 1.0 / (tau * gam * (w2 + 1j * k * v) + 1)
    c1 = -g2 / (g1 - g2)
    c2 = 1.0 - c1
    exact = c1 * np.exp(w1 * t) + c2 * np.exp(w2 * t)
    ratio = a1 / a0
    assert abs(np.angle(ratio) - np.angle(exact)) < 0.08 * abs(np.angle(exact))          # phase of the ripple
    # (without the d_0 alpha part the ripple of the rest-frame density lags behind the fluid: the covariant equation
    # would give the phase -k v t; the two are far apart, so the pin tells them apart)
    assert abs(np.angle(ratio) + k * v * t) > 0.3 * k * v * t
    assert abs((1 - abs(ratio)) / (1 - abs(exact)) - 1) < 0.12                            # as the static telegraph pin
    # the same run with the fluid at rest decays differently: time dilation and the projector are resolved
    disc = np.sqrt(complex(1 - 4 * tau * D * k * k))
    l1, l2 = (1 + disc) / (2 * tau), (1 - disc) / (2 * tau)
    rest = (-l2 / (l1 - l2) * np.exp(-l1 * t) + l1 / (l1 - l2) * np.exp(-l2 * t)).real
    assert abs((1 - abs(exact)) / (1 - rest) - 1) > 0.2


# -------------------------------------------------------------------------- energy in hyperbolic coordinates ----
def test_hyperbolic_energy_and_work_2d():
    """§5.6.5 (:1049-1063), reading 14, (2+1)D hyperbolic: E = sum (m/sigma*) tau T^{tau tau} is the energy per unit
    rapidity and nabla_mu T^{mu tau} = 0 gives dE/dtau = -sum (m/sigma*) tau^2 T^{eta eta} with tau^2 T^{eta eta} =
    p + Pi + tau^2 pi^{eta eta} (u^eta = 0) for the whole system, edges and transverse flow included.  Checked: the
    centred difference of E against that sum built from the read fields (O(dtau^2)); the WORK state field integrates
    exactly that sum, so E + work is conserved to the integration error, which shrinks with dtau."""
    n, dx, h, tau0 = 30, 0.1, 0.3, 0.6
    T0 = 0.30 / W.HBARC
    f = _slab(2, n, dx, tau0, T0)
    res = []
    for dt, ns in ((0.02, 8), (0.01, 16)):
        p = W.base_params(dim=2, coords=1, eom=1, flags=3, eos_kind=0, h=h, x0_start=tau0, dx0=dt, eta_over_s=0.2,
                          zeta_max=0.1, tau_Pi_coeff=1.0)
        o = O.Oracle(**p)
        o.load_particles(f)
        o.step(ns // 2 - 1)
        ta = o.conserved_totals()
        o.step(1)
        tb = o.conserved_totals()
        g = o.read_fields([O.P, O.BULK, O.PI33, O.SIGMA, O.SIGMA_STAR])
        taub = tb[0]
        rate = -np.sum((1.0 / g[O.SIGMA_STAR]) * (g[O.P] + g[O.BULK] * g[O.SIGMA] + taub ** 2 * g[O.PI33] * g[O.SIGMA]))
        o.step(1)
        tc = o.conserved_totals()
        dE = (tc[1] - ta[1]) / (tc[0] - ta[0])
        o.step(ns - ns // 2 - 1)
        td = o.conserved_totals()
        res.append((abs(dE / rate - 1), abs((td[1] + td[10]) / (ta[1] + ta[10]) - 1), tb[1]))
        # the per-particle work rate the integrator sees is the summand above
        wr = o.read_fields([O.RATE + O.WORK, O.P, O.BULK, O.PI33, O.SIGMA, O.SIGMA_STAR])
        exp = (1.0 / wr[O.SIGMA_STAR]) * (wr[O.P] + wr[O.BULK] * wr[O.SIGMA] + td[0] ** 2 * wr[O.PI33] * wr[O.SIGMA])
        assert np.allclose(wr[O.RATE + O.WORK], exp, rtol=1e-12)
    assert res[0][0] < 2e-3 and res[1][0] < 0.3 * res[0][0] + 1e-6       # O(dtau^2) centred difference
    assert res[0][1] < 2e-5 and res[1][1] < 2e-5                          # E + work conserved (the work alone is 6 % of E)
    # the value: uniform slab at rest, E = tau eps x (sum of particle volumes)
    assert res[1][2] > 0


def _static_fluid_hyperbolic(n, ne, dx, de, tau0, T0):
    """A uniform fluid at rest in (t, x, y, z), described in (tau, x, y, eta_s): u^tau = cosh eta, u^eta = -sinh eta / tau."""
    x1 = (np.arange(n) - 0.5 * (n - 1)) * dx
    e1 = (np.arange(ne) - 0.5 * (ne - 1)) * de
    X, Y, E = np.meshgrid(x1, x1, e1, indexing="ij")
    x, y, e = X.ravel(), Y.ravel(), E.ravel()
    gam = np.cosh(e)
    return {O.R1: x, O.R2: y, O.R3: e, O.U3: -np.sinh(e) / tau0, O.S: 4 * C0 * T0 ** 3 * gam * tau0 * dx * dx * de}


def test_hyperbolic_energy_3d_static_fluid():
    """Reading 14, (3+1)D: E = sum (m/sigma*) tau (T^{tau tau} cosh eta + tau T^{tau eta} sinh eta) is the Cartesian energy
    through the surface tau = const.  For a fluid at rest in the laboratory u^tau = cosh eta, u^eta = -sinh eta / tau and
    T^{tau tau} cosh eta + tau T^{tau eta} sinh eta = eps cosh eta identically, so E = tau sum_a (m/sigma*)_a eps_a cosh eta_a
    (to round-off; without the T^{tau eta} term it would be w cosh^3 - p cosh).  The fluid stays at rest: along a
    worldline z = tau sinh eta = const one has du^eta/dtau = 2 sinh eta / tau^2 and du^x/dtau = 0 (closed form for the
    (3+1)D momentum equation with u^eta != 0), and E stays constant while the interior is undisturbed."""
    n, ne, dx, de, tau0, h = 15, 19, 0.15, 0.15, 1.2, 0.3
    T0 = 0.30 / W.HBARC
    f = _static_fluid_hyperbolic(n, ne, dx, de, tau0, T0)
    p = W.base_params(dim=3, coords=1, eom=0, eos_kind=0, h=h, x0_start=tau0, dx0=0.01)
    o = O.Oracle(**p)
    o.load_particles(f)
    g = o.read_fields([O.E, O.SIGMA_STAR, O.RATE + O.U1, O.RATE + O.U3, O.T])
    t0 = o.conserved_totals()
    Eexp = tau0 * np.sum(g[O.E] / g[O.SIGMA_STAR] * np.cosh(f[O.R3]))
    assert abs(t0[1] / Eexp - 1) < 1e-12
    wrong = tau0 * np.sum((4.0 / 3.0 * g[O.E] * np.cosh(f[O.R3]) ** 3 - g[O.E] / 3.0 * np.cosh(f[O.R3])) / g[O.SIGMA_STAR])
    assert abs(wrong / Eexp - 1) > 0.3
    m = (np.abs(f[O.R1]) < 0.3) & (np.abs(f[O.R2]) < 0.3) & (np.abs(f[O.R3]) < 0.65)
    assert np.abs(g[O.T][m] / T0 - 1).max() < 1e-2 and np.ptp(g[O.T][m]) < 1e-3 * T0     # uniform (lattice sum error 0.5 %)
    exp3 = 2 * np.sinh(f[O.R3]) / tau0 ** 2
    assert np.abs(g[O.RATE + O.U3][m] - exp3[m]).max() < 0.01 * np.abs(exp3[m]).max()
    assert np.abs(g[O.RATE + O.U1][m]).max() < 0.01 * np.abs(exp3[m]).max()
    o.step(6)
    t1 = o.conserved_totals()
    assert abs(t1[1] / t0[1] - 1) < 2e-3
    # symmetric slab: no net longitudinal momentum develops
    assert abs(t1[4]) < 1e-9 * t0[1]


# ------------------------------------------------------------------------------------- (div v) accumulator ----
@pytest.mark.parametrize("D,coords", [(2, 0), (3, 1)])
def test_divv_is_minus_dlog_sigma_star_dt(D, coords):
    """Step 5, expansion rate: (div v)_a = (1/sigma*_a) sum_b m_b (v_b - v_a).grad W_ab is accumulated from v = u/gamma so
    that sigma*_a (div v)_a = -d sigma*_a/dx0 identically (Eq. 72 :882 differentiated along the particle paths).
    Finite difference of the oracle's own sigma* under x -> x +- v Delta (velocities frozen), random cloud, unequal
    masses."""
    rng = np.random.default_rng(5 + D)
    ns, dx, tau0 = (14, 0.15, 0.9) if D == 2 else (9, 0.15, 0.9)
    x1 = (np.arange(ns) - 0.5 * (ns - 1)) * dx
    g = np.meshgrid(*([x1] * D), indexing="ij")
    N = g[0].size
    pos = [g[k].ravel() + rng.uniform(-0.03, 0.03, N) for k in range(D)]
    u = [rng.normal(0, 0.4, N) for _ in range(D)]
    G = [1.0, 1.0, tau0 ** 2 if coords == 1 else 1.0]
    gam = np.sqrt(1 + sum(G[k] * u[k] ** 2 for k in range(D)))
    base = {O.S: rng.uniform(20, 60, N) * dx ** D, O.MASS: rng.uniform(0.8, 1.2, N)}
    for k in range(D):
        base[O.U1 + k] = u[k]
    p = W.base_params(dim=D, coords=coords, eom=0, eos_kind=0, h=0.3, x0_start=tau0, dx0=0.01)

    def sigma_star(shift):
        f = dict(base)
        for k in range(D):
            f[O.R1 + k] = pos[k] + shift * u[k] / gam
        o = O.Oracle(**p)
        o.load_particles(f)
        return o.read_fields([O.SIGMA_STAR, O.DIVV])
    r0 = sigma_star(0.0)
    d = 1e-4
    rp, rm = sigma_star(d)[O.SIGMA_STAR], sigma_star(-d)[O.SIGMA_STAR]
    lhs = (rp - rm) / (2 * d)
    rhs = -r0[O.SIGMA_STAR] * r0[O.DIVV]
    assert np.abs(rhs).max() > 1.0
    assert np.abs(lhs - rhs).max() < 1e-6 * np.abs(rhs).max()
