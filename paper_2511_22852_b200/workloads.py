"""Seeded synthetic inputs shaped like the paper's workloads (DESIGN.md §"Input recipe").

This module serves BOTH the CUDA library and the CPU oracle and therefore holds none of the method's
arithmetic (no SPH sums, no equations of motion, no table interpolation).  It only produces inputs:

  * analytic initial profiles (ideal Gubser flow, Eq. 116-120 :1137-1153; seeded hotspot events that
    stand in for the TRENTO/AMPT/ICCING events of PAPER.md §4, which are not available offline),
  * the offline-inverted equation-of-state table of the analytic conformal BSQ pressure (PAPER.md :583-593,
    App. A) — the "offline inverter" runs before the hot path and its output is an input of both sides,
  * the parameter sets of the five BASELINE.json configs (C1..C5) plus reduced variants used by the tests.

Everything is numpy; every random draw comes from numpy.random.Generator(PCG64(seed)) in a fixed order.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

HBARC = 0.1973269804  # GeV fm
SEED0 = 251122852

# state field ids (numeric convention of include/ccake.h and oracle/oracle.h)
R1, R2, R3, U1, U2, U3, S, NB, NS, NQ, BULK = range(11)
PI11, PI12, PI13, PI22, PI23, PI33 = range(11, 17)
JB1 = 17
MASS, WORK = 26, 27
# EoS table column ids
COL_T, COL_MUB, COL_MUS, COL_MUQ, COL_P, COL_CS2, COL_E, COL_WS, COL_WB, COL_WSQ, COL_WQ = range(11)

EOS_C0, EOS_C2, EOS_C4 = 5.26, 0.5, 0.05

KAPPA_OVER_T2 = [0.0482, -0.0482, 0.0, -0.0482, 0.1447, 0.0147, 0.0, 0.0147, 0.0880]
TAU_Q_TIMES_T = [0.2, 0.2, 0.2]
DNMR_DEFAULT = [2.0 / 3.0, 0.0, 4.0 / 3.0, 10.0 / 7.0, 6.0 / 5.0, 1.0, 0.0, 0.0]


@dataclass
class Workload:
    name: str
    params: dict
    fields: dict          # field id -> float64 array (length N)
    table: dict | None    # {"axes": [4 arrays], "axis_kind": [4], "col_ids": [...], "data": ndarray} or None
    nsteps: int
    meta: dict = field(default_factory=dict)

    @property
    def n(self) -> int:
        return len(next(iter(self.fields.values())))


def base_params(**kw) -> dict:
    p = dict(dim=2, coords=0, integrator=2, eom=0, flags=0, eos_kind=0, h=0.3, x0_start=1.0, dx0=0.05,
             eos_c0=EOS_C0, eos_c2=EOS_C2, eos_c4=EOS_C4, eta_over_s=0.0, tau_pi_coeff=5.0, tau_floor=0.005,
             zeta_max=0.0, zeta_T_peak=0.18 / HBARC, zeta_width=0.04 / HBARC, tau_Pi_coeff=1.0,
             kappa_over_T2=[0.0] * 9, tau_q_times_T=list(TAU_Q_TIMES_T), dnmr_coeffs=list(DNMR_DEFAULT))
    p.update(kw)
    return p


# ---------------------------------------------------------------------------------------------------- Gubser --
def gubser_T(tau, r, q=1.0, That0=None, T_center=0.4 / HBARC, tau0=1.0):
    """Ideal Gubser temperature, Eq. 116-118 with H0 = 0: T = (That0/tau) / cosh(rho)^(2/3),
    cosh^2 rho = [1 + 2 q^2 (tau^2 + r^2) + q^4 (tau^2 - r^2)^2] / (2 q tau)^2.
    That0 is fixed by T(tau0, 0) = T_center when not given."""
    def shape(t, rr):
        den = 1.0 + 2.0 * q * q * (t * t + rr * rr) + q ** 4 * (t * t - rr * rr) ** 2
        return (2.0 * q * t) ** (2.0 / 3.0) / (t * den ** (1.0 / 3.0))
    if That0 is None:
        That0 = T_center / shape(tau0, 0.0)
    return That0 * shape(np.asarray(tau, dtype=np.float64), np.asarray(r, dtype=np.float64))


def gubser_ur(tau, r, q=1.0):
    """Eq. 120."""
    den = np.sqrt(1.0 + 2.0 * q * q * (tau * tau + r * r) + q ** 4 * (tau * tau - r * r) ** 2)
    return 2.0 * q * q * r * tau / den


def shifted_gubser(tau, x, y, eta, t0=0.5, q=1.0, T_center=0.4 / HBARC, tau0=1.0):
    """Shifted Gubser solution, Eq. 113-125 (ideal).  Returns T, u^x, u^y, u^eta."""
    r = np.sqrt(x * x + y * y)
    taup = np.sqrt(tau * tau + 2.0 * t0 * tau * np.cosh(eta) + t0 * t0)
    T = gubser_T(taup, r, q=q, T_center=T_center, tau0=tau0)
    ur = gubser_ur(taup, r, q=q)
    den = np.sqrt(1.0 + 2.0 * q * q * (taup * taup + r * r) + q ** 4 * (taup * taup - r * r) ** 2)
    utau_p = (1.0 + q * q * (taup * taup + r * r)) / den
    with np.errstate(invalid="ignore", divide="ignore"):
        cx = np.where(r > 0, x / r, 0.0)
        cy = np.where(r > 0, y / r, 0.0)
    ueta = -utau_p * t0 * np.sinh(eta) / (tau * taup)
    return T, ur * cx, ur * cy, ueta


# ---------------------------------------------------------------------------------- conformal EoS (inputs) ----
def conformal_forward(T, mu, c0=EOS_C0, c2=EOS_C2, c4=EOS_C4):
    """p, s, n_q of p = c0 T^4 + c2 T^2 sum mu^2 + c4 sum mu^4 (an instance of Eq. A.5)."""
    mu = np.asarray(mu, dtype=np.float64)
    m2 = (mu ** 2).sum(axis=0)
    m4 = (mu ** 4).sum(axis=0)
    p = c0 * T ** 4 + c2 * T ** 2 * m2 + c4 * m4
    s = 4.0 * c0 * T ** 3 + 2.0 * c2 * T * m2
    n = 2.0 * c2 * T ** 2 * mu + 4.0 * c4 * mu ** 3
    return p, s, n


def conformal_invert_unit_s(yB, yS, yQ, c0=EOS_C0, c2=EOS_C2, c4=EOS_C4, iters=80):
    """(T, mu_q) at s = 1 and n_q = y_q (vectorised damped Newton on the 4 unknowns).  Because s and n_q are
    homogeneous of degree 3 in (T, mu), the solution at any s is s^(1/3) times this one."""
    y = np.stack([np.asarray(yB, np.float64), np.asarray(yS, np.float64), np.asarray(yQ, np.float64)])
    T = np.full(y.shape[1:], (1.0 / (4.0 * c0)) ** (1.0 / 3.0))
    mu = y / (2.0 * c2 * T ** 2)
    for _ in range(iters):
        _, s, n = conformal_forward(T, mu, c0, c2, c4)
        fs = s - 1.0
        fn = n - y
        m2 = (mu ** 2).sum(axis=0)
        Htt = 12.0 * c0 * T ** 2 + 2.0 * c2 * m2
        Htm = 4.0 * c2 * T * mu
        Hmm = 2.0 * c2 * T ** 2 + 12.0 * c4 * mu ** 2
        # Schur complement on the arrow matrix [[Htt, Htm^T], [Htm, diag(Hmm)]]
        schur = Htt - (Htm ** 2 / Hmm).sum(axis=0)
        dT = (fs - (Htm * fn / Hmm).sum(axis=0)) / schur
        dmu = (fn - Htm * dT) / Hmm
        T = T - dT
        mu = mu - dmu
    return T, mu


def log_decade_axis(n_nodes: int, per_decade: int, k0: int = -8):
    """s_{k,j} = 10^k (1 + 9 j / m): log-scaled overall, linearly spaced locally."""
    i = np.arange(n_nodes)
    return 10.0 ** (k0 + i // per_decade) * (1.0 + 9.0 * (i % per_decade) / per_decade)


def make_eos_table(ns=100, nq=32, ymax=0.05, with_wq=False, c0=EOS_C0, c2=EOS_C2, c4=EOS_C4):
    """Offline-inverted table on (s, rho_B/s, rho_S/s, rho_Q/s); columns T, mu_B, mu_S, mu_Q, p, cs2, e, dw/ds
    (+ dw/dn_q when with_wq).  Node values are the exact inversion of the analytic conformal pressure."""
    per_decade = 9 if ns <= 100 else 18
    s_ax = log_decade_axis(ns, per_decade)
    y_ax = np.linspace(-ymax, ymax, nq)
    YB, YS, YQ = np.meshgrid(y_ax, y_ax, y_ax, indexing="ij")
    T1, mu1 = conformal_invert_unit_s(YB, YS, YQ, c0, c2, c4)
    p1, s1, n1 = conformal_forward(T1, mu1, c0, c2, c4)
    assert np.max(np.abs(s1 - 1.0)) < 1e-12 and np.max(np.abs(n1 - np.stack([YB, YS, YQ]))) < 1e-12
    ncols = 11 if with_wq else 8
    data = np.empty((ns, nq, nq, nq, ncols), dtype=np.float64)
    s13 = np.cbrt(s_ax)[:, None, None, None]
    s43 = s13 ** 4
    data[..., COL_T] = s13 * T1
    data[..., COL_MUB] = s13 * mu1[0]
    data[..., COL_MUS] = s13 * mu1[1]
    data[..., COL_MUQ] = s13 * mu1[2]
    data[..., COL_P] = s43 * p1
    data[..., COL_CS2] = 1.0 / 3.0
    data[..., COL_E] = 3.0 * s43 * p1
    data[..., COL_WS] = (4.0 / 3.0) * s13 * T1           # conformal: H (T, mu) = 3 (s, n)  =>  dw/ds = 4T/3
    if with_wq:
        data[..., COL_WB] = (4.0 / 3.0) * s13 * mu1[0]
        data[..., COL_WSQ] = (4.0 / 3.0) * s13 * mu1[1]
        data[..., COL_WQ] = (4.0 / 3.0) * s13 * mu1[2]
    return dict(axes=[s_ax, y_ax, y_ax, y_ax], axis_kind=[0, 1, 1, 1], col_ids=list(range(ncols)), data=data)


def signed_geometric_axis(n: int, xmax: float, xmin: float):
    """n nodes: -xmax ... -xmin (geometric, n // 2 - 1 ... nodes), 0, +xmin ... +xmax (geometric): log-scaled on both sides
    of zero, as (T, mu) tables that have to serve many decades of temperature are."""
    nneg = (n - 1) // 2
    npos = n - 1 - nneg
    return np.concatenate([-np.geomspace(xmax, xmin, nneg), [0.0], np.geomspace(xmin, xmax, npos)])


def make_forward_table(nT=100, nmu=32, T_lo=5e-4, T_hi=4.0, mu_lo=1e-5, mu_hi=4.4, c0=EOS_C0, c2=EOS_C2, c4=EOS_C4):
    """Input of the offline inverter (BASELINE.json configs[1]: "tabulated forward on a 100x32x32x32 (T, mu_B, mu_S, mu_Q)
    grid"): (p, s, n_B, n_S, n_Q) of the analytic conformal BSQ pressure at the nodes of a geometric T axis and three
    signed-geometric mu axes.  Returns dict(axes=[T, mu, mu, mu], data[nT, nmu, nmu, nmu, 5])."""
    T_ax = np.geomspace(T_lo, T_hi, nT)
    m_ax = signed_geometric_axis(nmu, mu_hi, mu_lo)
    T, mB, mS, mQ = np.meshgrid(T_ax, m_ax, m_ax, m_ax, indexing="ij")
    p, s, n = conformal_forward(T, np.stack([mB, mS, mQ]), c0, c2, c4)
    data = np.stack([p, s, n[0], n[1], n[2]], axis=-1)
    return dict(axes=[T_ax, m_ax, m_ax, m_ax], data=np.ascontiguousarray(data))


# ------------------------------------------------------------------------------------------- Gubser configs ---
def _square_lattice(n, dx):
    x1 = (np.arange(n) - 0.5 * (n - 1)) * dx
    X, Y = np.meshgrid(x1, x1, indexing="xy")
    return X.ravel(), Y.ravel()


def config_c1(hyperbolic=False, n=50, dx=0.2, nsteps=20, dt=0.05, integrator=2):
    """C1: (2+1)D ideal conformal fluid, closed-form EoS; Cartesian (u = 0) or, as C1h, hyperbolic Gubser."""
    x, y = _square_lattice(n, dx)
    r = np.hypot(x, y)
    T = gubser_T(1.0, r)
    s = 4.0 * EOS_C0 * T ** 3
    if hyperbolic:
        ur = gubser_ur(1.0, r)
        with np.errstate(invalid="ignore", divide="ignore"):
            ux = np.where(r > 0, ur * x / r, 0.0)
            uy = np.where(r > 0, ur * y / r, 0.0)
        gam = np.sqrt(1.0 + ux ** 2 + uy ** 2)
        sqrtg = 1.0
    else:
        ux = np.zeros_like(x)
        uy = np.zeros_like(x)
        gam = np.ones_like(x)
        sqrtg = 1.0
    tau0 = 1.0
    if hyperbolic:
        sqrtg = tau0
    fields = {R1: x, R2: y, U1: ux, U2: uy, S: s * gam * sqrtg * dx * dx}
    params = base_params(dim=2, coords=1 if hyperbolic else 0, integrator=integrator, eom=0, eos_kind=0, h=0.3,
                         x0_start=tau0, dx0=dt)
    return Workload("C1h" if hyperbolic else "C1", params, fields, None, nsteps, dict(dx=dx, n_side=n))


def config_c2(n=200, dx=0.1, nsteps=50, dt=0.05, ns=100, nq=32, mu_over_T=0.1, table=None):
    """C2: (2+1)D ideal BSQ Gubser, hyperbolic, EoS table 100x32^3 with 8 columns."""
    x, y = _square_lattice(n, dx)
    r = np.hypot(x, y)
    tau0 = 1.0
    T = gubser_T(tau0, r)
    mu = np.stack([mu_over_T * T] * 3)
    _, s, nq_ = conformal_forward(T, mu)
    ur = gubser_ur(tau0, r)
    with np.errstate(invalid="ignore", divide="ignore"):
        ux = np.where(r > 0, ur * x / r, 0.0)
        uy = np.where(r > 0, ur * y / r, 0.0)
    gam = np.sqrt(1.0 + ux ** 2 + uy ** 2)
    vol = gam * tau0 * dx * dx
    fields = {R1: x, R2: y, U1: ux, U2: uy, S: s * vol, NB: nq_[0] * vol, NS: nq_[1] * vol, NQ: nq_[2] * vol}
    params = base_params(dim=2, coords=1, eom=0, eos_kind=1, h=0.3, x0_start=tau0, dx0=dt)
    if table is None:
        table = make_eos_table(ns=ns, nq=nq, with_wq=False)
    return Workload("C2", params, fields, table, nsteps, dict(dx=dx, n_side=n, mu_over_T=mu_over_T))


# --------------------------------------------------------------------------------------- hotspot event tiles --
def _woods_saxon_radius(rng, R, a):
    rmax = R + 10.0 * a
    rr = np.linspace(0.0, rmax, 4001)
    fmax = float(np.max(rr * rr / (1.0 + np.exp((rr - R) / a))))
    while True:
        r = rng.uniform(0.0, rmax)
        v = rng.uniform(0.0, 1.0)
        if v * fmax < r * r / (1.0 + math.exp((r - R) / a)):
            return r


def _event_tile(seed, tile, n_side, dx, n_hot, width, R, a, eta_nodes=None, stopping=False,
                T_peak=0.45 / HBARC, T_bg=0.05 / HBARC, rq=(0.005, 0.002, 0.0025)):
    """One seeded event on an n_side^2 (x n_eta) lattice; returns positions (tile-local), s, rho_q (rest frame).
    Draw order per hotspot: radius (rejection), cos(theta), phi, amplitude, u_B, u_S, u_Q."""
    rng = np.random.Generator(np.random.PCG64(seed + 1000 * tile))
    xs = np.empty(n_hot); ys = np.empty(n_hot); A = np.empty(n_hot); uq = np.empty((n_hot, 3))
    for k in range(n_hot):
        r = _woods_saxon_radius(rng, R, a)
        ct = rng.uniform(-1.0, 1.0)
        ph = rng.uniform(0.0, 2.0 * math.pi)
        st = math.sqrt(max(0.0, 1.0 - ct * ct))
        xs[k] = r * st * math.cos(ph)
        ys[k] = r * st * math.sin(ph)
        A[k] = math.exp(0.5 * rng.standard_normal())
        uq[k] = rng.uniform(-1.0, 1.0, size=3)
    x1 = (np.arange(n_side) - 0.5 * (n_side - 1)) * dx
    X, Y = np.meshgrid(x1, x1, indexing="xy")
    ehot = np.zeros_like(X)
    wq = np.zeros((3,) + X.shape)
    for k in range(n_hot):
        gk = A[k] * np.exp(-((X - xs[k]) ** 2 + (Y - ys[k]) ** 2) / (2.0 * width * width))
        ehot += gk
        for q in range(3):
            wq[q] += gk * (1.0 + 0.2 * uq[k, q])
    with np.errstate(invalid="ignore", divide="ignore"):
        fq = np.where(ehot > 1e-300, wq / np.maximum(ehot, 1e-300), 1.0)
    e_peak = 3.0 * EOS_C0 * T_peak ** 4
    e_bg = 3.0 * EOS_C0 * T_bg ** 4
    if eta_nodes is None:
        prof = ehot / ehot.max()
        eps = e_bg + (e_peak - e_bg) * prof
        s = 4.0 * EOS_C0 * (eps / (3.0 * EOS_C0)) ** 0.75
        rho = np.stack([rq[q] * s * fq[q] for q in range(3)])
        return X.ravel(), Y.ravel(), None, s.ravel(), rho.reshape(3, -1)
    eta = np.asarray(eta_nodes, dtype=np.float64)
    feta = np.where(np.abs(eta) < 2.0, 1.0, np.exp(-0.5 * (np.abs(eta) - 2.0) ** 2))
    e3 = ehot[None, :, :] * feta[:, None, None]
    prof = e3 / e3.max()
    eps = e_bg + (e_peak - e_bg) * prof
    s = 4.0 * EOS_C0 * (eps / (3.0 * EOS_C0)) ** 0.75
    rho = np.stack([rq[q] * s * fq[q][None, :, :] for q in range(3)])
    if stopping:   # baryon stopping at both beam rapidities (config 5)
        stop = np.exp(-(eta - 1.5) ** 2 / 0.5) + np.exp(-(eta + 1.5) ** 2 / 0.5)
        rho[0] = rho[0] * stop[:, None, None] * 4.0
    X3 = np.broadcast_to(X[None], e3.shape)
    Y3 = np.broadcast_to(Y[None], e3.shape)
    E3 = np.broadcast_to(eta[:, None, None], e3.shape)
    return X3.ravel(), Y3.ravel(), E3.ravel(), s.ravel(), rho.reshape(3, -1)


def _tiled_event(name, cfg_index, K, n_side, dx, n_hot, width, R, a, params, nsteps, eta_nodes=None,
                 stopping=False, table=None, tile0=0):
    h = params["h"]
    gap = 2.0 * h + 2.0 * nsteps * params["dx0"]
    box = n_side * dx
    wide = int(math.ceil(math.sqrt(K)))
    cols = {R1: [], R2: [], R3: [], S: [], NB: [], NS: [], NQ: []}
    tau0 = params["x0_start"] if params["coords"] == 1 else 1.0
    dV = dx * dx * ((eta_nodes[1] - eta_nodes[0]) if eta_nodes is not None else 1.0)
    for t in range(K):
        x, y, e, s, rho = _event_tile(SEED0 + cfg_index, tile0 + t, n_side, dx, n_hot, width, R, a, eta_nodes, stopping)
        ox = (t % wide) * (box + gap)
        oy = (t // wide) * (box + gap)
        cols[R1].append(x + ox); cols[R2].append(y + oy)
        if e is not None:
            cols[R3].append(e)
        vol = tau0 * dV          # gamma = 1: the event tiles start at rest (reading 10, 17)
        cols[S].append(s * vol)
        for q, fid in enumerate((NB, NS, NQ)):
            cols[fid].append(rho[q] * vol)
    fields = {k: np.concatenate(v) for k, v in cols.items() if v}
    deta = float(eta_nodes[1] - eta_nodes[0]) if eta_nodes is not None else 1.0
    return Workload(name, params, fields, table, nsteps, dict(tiles=K, n_side=n_side, dx=dx, gap=gap, deta=deta))


def viscous_params(dim, eom, dx0, x0=0.6):
    return base_params(dim=dim, coords=1, eom=eom, flags=7, eos_kind=1, h=0.3, x0_start=x0, dx0=dx0,
                       eta_over_s=0.08, tau_pi_coeff=5.0, tau_floor=0.005, zeta_max=0.1,
                       zeta_T_peak=0.18 / HBARC, zeta_width=0.04 / HBARC, tau_Pi_coeff=1.0,
                       kappa_over_T2=list(KAPPA_OVER_T2), tau_q_times_T=list(TAU_Q_TIMES_T))


def config_c3(K=4, n_side=233, nsteps=100, n_hot=200, table=None, tile0=0):
    """C3: (2+1)D viscous Pb+Pb-like event tiles, minimal IS shear + bulk + BSQ diffusion, 11-column table."""
    params = viscous_params(2, 1, 0.025)
    if table is None:
        table = make_eos_table(100, 32, with_wq=True)
    return _tiled_event("C3", 3, K, n_side, 0.06, n_hot, 0.5, 6.6, 0.45, params, nsteps, table=table, tile0=tile0)


def config_c4(K=10, n_side=80, n_eta=31, nsteps=50, n_hot=40, table=None, tile0=0):
    """C4: (3+1)D viscous O+O-like event tiles, DNMR shear + bulk + diffusion, 11-column table."""
    params = viscous_params(3, 2, 0.05)
    eta = (np.arange(n_eta) - 0.5 * (n_eta - 1)) * 0.1
    if table is None:
        table = make_eos_table(100, 32, with_wq=True)
    return _tiled_event("C4", 4, K, n_side, 0.1, n_hot, 0.4, 2.6, 0.513, params, nsteps, eta_nodes=eta, table=table,
                        tile0=tile0)


def config_c4p(n_side=126, spacing=0.2244, nsteps=10, n_hot=40, table=None):
    """C4': the sparse throughput probe — C4's physics and generator stretched to a simple cubic
    lattice of n_side^3 sites with spacing 0.2244 in x, y and eta_s (2,000,376 particles, ~80 neighbours at h = 0.3 fm):
    the regime BASELINE.json's config 4 states ("~80 neighbours"), where the substep sits near the HBM / FP64 ridge."""
    params = viscous_params(3, 2, 0.05)
    stretch = n_side * spacing / 8.0
    eta = (np.arange(n_side) - 0.5 * (n_side - 1)) * spacing
    if table is None:
        table = make_eos_table(100, 32, with_wq=True)
    w = _tiled_event("C4p", 6, 1, n_side, spacing, n_hot, 0.4 * stretch, 2.6 * stretch, 0.513 * stretch, params, nsteps,
                     eta_nodes=eta / stretch * 1.0, table=table)
    # the rapidity profile of C4 (plateau half-width 2, Gaussian tails) is evaluated on eta / stretch; the lattice itself
    # has the cubic spacing
    f = dict(w.fields)
    f[R3] = np.tile(np.repeat(eta, n_side * n_side), 1)
    vol_fix = spacing / ((eta[1] - eta[0]) / stretch)
    for k in (S, NB, NS, NQ):
        f[k] = f[k] * vol_fix
    meta = dict(w.meta)
    meta["deta"] = spacing
    return Workload("C4p", params, f, table, nsteps, meta)


def config_c5(K=13, n_side=266, n_eta=21, nsteps=20, n_hot=400, table=None, ns=200, nq=48, tile0=0):
    """C5: (3+1)D high-resolution Au+Au-like event tiles with baryon stopping, minimal IS, 200x48^3 table."""
    params = viscous_params(3, 1, 0.025)
    eta = (np.arange(n_eta) - 0.5 * (n_eta - 1)) * 0.15
    if table is None:
        table = make_eos_table(ns, nq, with_wq=True)
    return _tiled_event("C5", 5, K, n_side, 0.06, n_hot, 0.5, 6.4, 0.54, params, nsteps, eta_nodes=eta,
                        stopping=True, table=table, tile0=tile0)


def with_dissipative_state(w: Workload, seed: int, amp: float = 0.03, u_amp: float = 0.05) -> Workload:
    """The same workload with a seeded non-equilibrium start: velocities u^i ~ N(0, u_amp) and Pi/sigma, pi^{ij}/sigma,
    J^i_q/sigma drawn per particle as N(0, 1) times amp times the particle's equilibrium scale (energy per particle
    for Pi and pi, charge per particle for J; eta components carry 1/tau per index).  The event tiles of C3-C5 start
    at rest with Pi = pi = J = 0 (reading 17), where every second-order coupling multiplies numbers near zero; this
    variant exercises them in the same launch configuration.  Draw order: u (per component), Pi, pi (11, 12, 22, 33,
    13, 23), J (q-major)."""
    p = w.params
    D, tau0 = p["dim"], (p["x0_start"] if p["coords"] == 1 else 1.0)
    rng = np.random.Generator(np.random.PCG64(SEED0 + 7919 * seed))
    f = dict(w.fields)
    n = w.n
    dxyz = w.meta.get("dx", 0.1)
    vol = tau0 * dxyz ** 2 * (w.meta.get("deta", 0.1) if D == 3 else 1.0)
    s = f[S] / vol
    T = np.cbrt(s / (4.0 * EOS_C0))
    escale = 3.0 * EOS_C0 * T ** 4 * vol
    gfac = [1.0, 1.0, 1.0 / tau0 if p["coords"] == 1 else 1.0]
    for k in range(D):
        f[U1 + k] = u_amp * rng.standard_normal(n) * gfac[k]
    f[BULK] = amp * escale * rng.standard_normal(n)
    comps = [(PI11, 0, 0), (PI12, 0, 1), (PI22, 1, 1), (PI33, 2, 2)] + ([(PI13, 0, 2), (PI23, 1, 2)] if D == 3 else [])
    for fid, i, j in comps:
        f[fid] = amp * escale * rng.standard_normal(n) * gfac[i] * gfac[j]
    for q in range(3):
        for k in range(D):
            f[JB1 + 3 * q + k] = amp * np.abs(f[NB + q]) * rng.standard_normal(n) * gfac[k]
    return Workload(w.name + "_neq", p, f, w.table, w.nsteps, dict(w.meta))


def count_pairs_estimate(w: Workload) -> float:
    """Continuum estimate of ordered neighbour pairs per pass, Eq. 132-133 (for sizing only)."""
    p = w.params
    dx = w.meta.get("dx", 0.1)
    if p["dim"] == 2:
        return w.n * math.pi * (2 * p["h"]) ** 2 / dx ** 2
    return w.n * 4.0 / 3.0 * math.pi * (2 * p["h"]) ** 3 / (dx * dx * 0.1)
