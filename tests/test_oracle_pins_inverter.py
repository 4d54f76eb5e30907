"""Pins of the oracle's offline inverter on a TABULATED forward EoS (PAPER.md :576-593, DESIGN reading 21), -m "not gpu".

`oracle_invert_forward_table` is an iteration (damped Newton on a quadrilinear interpolant), so the oracle follows the
algorithm of reading 21 step by step; these tests pin it to things other than itself:
  * an affine forward map, where interpolation is exact and the answer is numpy's linear solve (non-symmetric matrix,
    so a transposed Jacobian fails),
  * scipy's RegularGridInterpolator (an independent multilinear interpolator) for the round trip,
  * the exact closed-form inversion of the conformal BSQ EoS (App. A), approached at second order as the forward grid
    is refined,
  * the backup EoS (:572) for targets the table cannot reach.
"""
import numpy as np
import pytest
from scipy.interpolate import RegularGridInterpolator

import oracle as O
from paper_2511_22852_b200 import workloads as W

C0, C2, C4 = W.EOS_C0, W.EOS_C2, W.EOS_C4


def _params():
    return O.make_params(dim=2, coords=0, integrator=2, eom=0, flags=0, eos_kind=0, h=0.3, x0_start=0.0, dx0=0.05,
                         eos_c0=C0, eos_c2=C2, eos_c4=C4)


def _conformal_forward(T, mu):
    """App. A Eq. A.5-A.7 (:2115-2122): p, s = dp/dT, n_q = dp/dmu_q of p = c0 T^4 + c2 T^2 sum mu^2 + c4 sum mu^4."""
    m2 = sum(m * m for m in mu)
    m4 = sum(m ** 4 for m in mu)
    p = C0 * T ** 4 + C2 * T * T * m2 + C4 * m4
    s = 4 * C0 * T ** 3 + 2 * C2 * T * m2
    n = [2 * C2 * T * T * m + 4 * C4 * m ** 3 for m in mu]
    return p, s, n


def _forward_table(axes, fn):
    g = np.meshgrid(*axes, indexing="ij")
    p, s, n = fn(g[0], [g[1], g[2], g[3]])
    return np.stack([p, s, n[0], n[1], n[2]], axis=-1)


def test_affine_forward_map_is_inverted_exactly():
    """Interpolation of an affine map is exact, so the root is X = A^-1 (Y* - b) and every derived column has a closed
    form in A: z = A^-T Y*, c_s^2 = Y*.A^-1 Y* / X.Y*, e = T s - p + mu.n (reading 21)."""
    rng = np.random.default_rng(7)
    A = np.array([[3.0, 0.4, -0.2, 0.1], [0.3, 2.0, 0.5, -0.3], [-0.1, 0.2, 1.5, 0.6], [0.25, -0.4, 0.1, 1.8]])
    b = np.array([5.0, 0.3, -0.2, 0.1])
    cp, dp = np.array([0.7, 0.2, -0.1, 0.3]), 0.4
    axes = [np.linspace(0.5, 2.0, 7), np.linspace(-1.0, 1.0, 5), np.linspace(-0.8, 1.2, 6), np.sort(rng.uniform(-1, 1, 5))]
    g = np.stack(np.meshgrid(*axes, indexing="ij"), axis=-1)
    Y = g @ A.T + b
    fdata = np.concatenate([(g @ cp + dp)[..., None], Y], axis=-1)
    Xt = np.stack([rng.uniform(a[0], a[-1], 50) for a in axes], axis=1)
    Yt = Xt @ A.T + b
    out, flag, iters = O.invert_forward_table(_params(), axes, fdata, Yt[:, 0], [Yt[:, 1], Yt[:, 2], Yt[:, 3]])
    assert np.all(flag == 0) and iters.max() <= 3
    X = np.linalg.solve(A, (Yt - b).T).T
    assert np.max(np.abs(X - Xt)) < 1e-12
    assert np.max(np.abs(out[:, 0:4] - X)) < 1e-12
    p = X @ cp + dp
    assert np.max(np.abs(out[:, 4] - p)) < 1e-12
    e = X[:, 0] * Yt[:, 0] - p + np.sum(X[:, 1:] * Yt[:, 1:], axis=1)
    assert np.max(np.abs(out[:, 6] - e)) < 1e-11
    z = np.linalg.solve(A.T, Yt.T).T
    assert np.max(np.abs(out[:, 7] - (X[:, 0] + z[:, 0]))) < 1e-11
    assert np.max(np.abs(out[:, 8:11] - (X[:, 1:] + z[:, 1:]))) < 1e-11
    v = np.linalg.solve(A, Yt.T).T
    cs2 = np.sum(Yt * v, axis=1) / np.sum(X * Yt, axis=1)
    assert np.max(np.abs(out[:, 5] - cs2)) < 1e-11


def _conformal_case(nT, nmu, seed=3, nt=200):
    axes = [np.linspace(0.1, 0.5, nT)] + [np.linspace(-0.3, 0.3, nmu)] * 3
    fdata = _forward_table(axes, _conformal_forward)
    rng = np.random.default_rng(seed)
    T = rng.uniform(0.15, 0.45, nt)
    mu = [rng.uniform(-0.25, 0.25, nt) for _ in range(3)]
    p, s, n = _conformal_forward(T, mu)
    return axes, fdata, T, mu, p, s, n


def test_round_trip_through_an_independent_interpolator():
    """The root X satisfies interp(X) = (s*, n*) for scipy's multilinear interpolator of the same table, and the
    pressure column is that interpolator's p(X)."""
    axes, fdata, T, mu, p, s, n = _conformal_case(17, 9)
    out, flag, _ = O.invert_forward_table(_params(), axes, fdata, s, n)
    assert np.all(flag == 0)
    X = out[:, 0:4]
    for c, want in [(1, s), (2, n[0]), (3, n[1]), (4, n[2])]:
        got = RegularGridInterpolator(axes, fdata[..., c])(X)
        assert np.max(np.abs(got - want) / s) < 1e-12
    assert np.max(np.abs(RegularGridInterpolator(axes, fdata[..., 0])(X) - out[:, 4])) < 1e-13


def test_target_at_a_node_returns_the_node():
    axes, fdata, *_ = _conformal_case(9, 5)
    idx = [(2, 1, 3, 2), (7, 3, 1, 1), (4, 2, 2, 2), (1, 3, 3, 1)]
    s = np.array([fdata[i][1] for i in idx])
    n = [np.array([fdata[i][2 + q] for i in idx]) for q in range(3)]
    out, flag, _ = O.invert_forward_table(_params(), axes, fdata, s, n)
    assert np.all(flag == 0)
    for k, i in enumerate(idx):
        want = [axes[a][i[a]] for a in range(4)]
        assert np.max(np.abs(out[k, 0:4] - want)) < 1e-11
        assert abs(out[k, 4] - fdata[i][0]) < 1e-12


def test_second_order_convergence_to_the_exact_conformal_inversion():
    """Refining the forward grid by 2 cuts the error of (T, mu, p, e) against the exact inversion (Eq. A.11-A.15 via the
    known (T, mu) the targets were made from) by ~4; the Jacobian-derived columns (c_s^2, dw/ds, dw/dn_q) converge too
    (first order: derivative of a piecewise multilinear interpolant)."""
    P = _params()
    errs, errs_d = [], []
    for nT, nmu in [(9, 7), (17, 13), (33, 25)]:
        axes, fdata, T, mu, p, s, n = _conformal_case(nT, nmu)
        out, flag, _ = O.invert_forward_table(P, axes, fdata, s, n)
        assert np.all(flag == 0)
        e = [np.max(np.abs(out[:, 0] - T)), max(np.max(np.abs(out[:, 1 + q] - mu[q])) for q in range(3)),
             np.max(np.abs(out[:, 4] - p) / p), np.max(np.abs(out[:, 6] - 3 * p) / p)]
        errs.append(e)
        exact = np.array([O.eos_closed_form(P, s[a], [n[q][a] for q in range(3)]) for a in range(len(s))])
        errs_d.append([np.max(np.abs(out[:, 5] - 1.0 / 3.0)), np.max(np.abs(out[:, 7] - exact[:, 7])),
                       np.max(np.abs(out[:, 8:11] - exact[:, 8:11]))])
    errs, errs_d = np.array(errs), np.array(errs_d)
    assert np.all(errs[0] / errs[1] > 3.0) and np.all(errs[1] / errs[2] > 3.0), errs
    assert np.all(errs[2] < [5e-4, 1e-3, 5e-3, 2e-2]), errs[2]
    assert np.all(errs_d[0] / errs_d[2] > 3.0), errs_d
    assert np.all(errs_d[2] < [0.04, 0.02, 0.05]), errs_d[2]


def test_unreachable_targets_take_the_backup_eos():
    """:572, :583: a target outside the image of the table falls to the backup EoS — here the closed-form conformal one
    of the parameters — and is flagged."""
    P = _params()
    axes, fdata, T, mu, p, s, n = _conformal_case(9, 7, nt=6)
    s2 = s.copy()
    s2[0] = 50.0 * fdata[..., 1].max()              # hotter than the table
    s2[1] = 1e-3 * fdata[..., 1].min()              # colder than the table
    n2 = [x.copy() for x in n]
    n2[0][2] = 10.0 * fdata[..., 2].max()           # denser than the table
    out, flag, _ = O.invert_forward_table(P, axes, fdata, s2, n2)
    assert list(flag) == [1, 1, 1, 0, 0, 0]
    for a in range(3):
        want = O.eos_closed_form(P, s2[a], [n2[q][a] for q in range(3)])
        assert np.array_equal(out[a], want)


def test_rejects_a_bad_axis():
    axes, fdata, T, mu, p, s, n = _conformal_case(5, 3, nt=2)
    axes[2] = axes[2][::-1].copy()
    with pytest.raises(O.OracleError):
        O.invert_forward_table(_params(), axes, fdata, s, n)
