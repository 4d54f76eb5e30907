"""Helpers shared by the -m gpu parity tests: build both sides from one seeded Workload and compare.

The CUDA library is reached only through its C ABI (paper_2511_22852_b200.binding -> libccake.so); the oracle only
through oracle/ (liboracle.so).  Tolerances (DESIGN.md §"Tolerances"):
  * integer work (cell ids, neighbour sets): bit-exact;
  * smoothed densities after one evaluation: 1e-11 relative, element-wise (sums of O(10^2..10^3) positive terms);
  * signed sums with cancellation (gradient sums, rates): 1e-10 of the field's infinity norm;
  * fields after k RK steps: 1e-8 norm-wise, and element-wise for the positive fields (sigma*, s, T, p).
"""
import numpy as np

import oracle as O
from paper_2511_22852_b200 import binding as B

TOL_SUM = 1e-11
TOL_GRAD = 1e-10
TOL_RUN = 1e-8

POSITIVE = (B.SIGMA_STAR, B.S_DENS, B.T, B.P, B.E, B.GAMMA, B.SIGMA, B.S_STAR)


def state_ids(params):
    D = params["dim"]
    ids = [B.R1, B.R2, B.U1, B.U2, B.S, B.NB, B.NS, B.NQ]
    if D == 3:
        ids += [B.R3, B.U3]
    fl = params["flags"] if params["eom"] != 0 else 0
    if fl & 2:
        ids.append(B.BULK)
    if fl & 1:
        ids += [B.PI11, B.PI12, B.PI22, B.PI33] + ([B.PI13, B.PI23] if D == 3 else [])
    if fl & 4:
        ids += [B.JB1 + 3 * q + j for q in range(3) for j in range(D)]
    if params["coords"] == 1 and D == 2:
        ids.append(B.WORK)
    return ids


def derived_ids(params):
    ids = [B.SIGMA_STAR, B.S_STAR, B.RHOSTAR_B, B.RHOSTAR_S, B.RHOSTAR_Q, B.SIGMA, B.S_DENS, B.RHO_B, B.RHO_S,
           B.RHO_Q, B.GAMMA, B.T, B.MU_B, B.MU_S, B.MU_Q, B.P, B.E, B.CS2, B.WS]
    return ids


def gradient_ids(params):
    D = params["dim"]
    return [B.DIVV, B.THETA] + [B.FM1 + k for k in range(D)] + [B.FK_B, B.FK_S, B.FK_Q]


def make_pair(w, memspace="host"):
    g = B.from_workload(w, memspace=memspace)
    o = O.Oracle(**w.params)
    if w.table is not None:
        o.load_eos_table(w.table["axes"], w.table["axis_kind"], w.table["col_ids"], w.table["data"])
    o.load_particles(w.fields)
    return g, o


def norm_rel(a, b):
    """||a - b||_inf / ||b||_inf (0 when both vanish)."""
    den = float(np.max(np.abs(b))) if b.size else 0.0
    num = float(np.max(np.abs(a - b))) if b.size else 0.0
    if den == 0.0:
        return 0.0 if num == 0.0 else np.inf
    return num / den


def elem_rel(a, b):
    with np.errstate(divide="ignore", invalid="ignore"):
        r = np.abs(a - b) / np.abs(b)
    r[(a == b)] = 0.0
    return float(np.max(r)) if r.size else 0.0


def assert_fields(g, o, ids, tol, what, elementwise=()):
    fg = g.read_fields(ids)
    fo = o.read_fields(ids)
    worst = {}
    for k in ids:
        assert np.all(np.isfinite(fg[k])), f"{what}: field {k} not finite on the GPU"
        e = elem_rel(fg[k], fo[k]) if k in elementwise else norm_rel(fg[k], fo[k])
        worst[k] = e
    bad = {k: v for k, v in worst.items() if not (v <= tol)}
    assert not bad, f"{what}: fields beyond {tol:g}: {bad}"
    return worst


def assert_neighbours_equal(g, o):
    cg, og, lg = g.read_neighbors()
    co, oo, lo = o.read_neighbors()
    assert np.array_equal(cg, co), "neighbour counts differ"
    assert np.array_equal(og, oo)
    assert np.array_equal(lg, lo), "neighbour lists differ"
    return int(co.sum())


def assert_cells_equal(g, o):
    a = g.read_fields([B.CELL])[B.CELL]
    b = o.read_fields([O.CELL])[O.CELL]
    assert np.array_equal(a, b), "reported cell ids differ"


def drift(t0, t1):
    """relative drift of E, S_tot and absolute drift of P_i, N_q between two ccake totals vectors"""
    return dict(E=abs(t1[1] + t1[10] - t0[1] - t0[10]) / abs(t0[1]), S=abs(t1[5] - t0[5]) / abs(t0[5]),
                P=float(np.max(np.abs(t1[2:5] - t0[2:5]))), N=float(np.max(np.abs(t1[6:9] - t0[6:9]))))
