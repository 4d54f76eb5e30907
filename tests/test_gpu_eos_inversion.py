"""NEXT-1 of SURVEY.md §8(f): the offline EoS inversion done on the device (ccake_invert_eos_table), against the
oracle's closed-form inversion (oracle_eos_closed_form, node by node) and against the host table generator."""
import numpy as np
import pytest

import oracle as O
from paper_2511_22852_b200 import binding as B
from paper_2511_22852_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _ctx():
    w = W.config_c1()
    p = dict(w.params)
    p["eos_kind"] = 1
    return B.Ccake(**p), O.make_params(**w.params)


def test_inverted_table_matches_oracle_node_by_node():
    """Every column at a seeded sample of nodes of a 100 x 12^3 grid (log-decade s axis, n_q / s axes), plus all
    nodes of the corner lines: 1e-12 relative (both sides bisect T to the last bit and solve the same cubic)."""
    g, P = _ctx()
    tb = W.make_eos_table(100, 12, with_wq=True)
    got = g.invert_eos_table(tb["axes"], tb["axis_kind"], tb["col_ids"], out=True)
    assert got.shape == tb["data"].shape and np.all(np.isfinite(got))
    rng = np.random.default_rng(2511)
    idx = [tuple(rng.integers(0, n) for n in got.shape[:4]) for _ in range(400)]
    idx += [(i, 0, 0, 0) for i in range(got.shape[0])] + [(i, 11, 11, 11) for i in range(got.shape[0])]
    ax = tb["axes"]
    for (i0, i1, i2, i3) in idx:
        s = ax[0][i0]
        n = [ax[1][i1] * s, ax[2][i2] * s, ax[3][i3] * s]
        ref = O.eos_closed_form(P, s, n)          # T, mu_B, mu_S, mu_Q, p, cs2, e, ws, wB, wS, wQ
        val = got[i0, i1, i2, i3]
        scale = np.array([ref[0]] * 4 + [ref[4], 1.0, ref[6], ref[0]] + [ref[0]] * 3)
        assert np.all(np.abs(val - ref) <= 1e-12 * np.abs(scale)), ((i0, i1, i2, i3), val, ref)
    g.close()


def test_inverted_table_equals_host_generator_and_drives_the_path():
    """The device-built table equals workloads.make_eos_table (which inverts by scaling a unit-s solution) to
    1e-10, and a run on it gives the same fields as a run on the loaded table."""
    tb = W.make_eos_table(100, 8, with_wq=False)
    w = W.config_c2(n=60, dx=0.1, nsteps=5, table=tb)
    g1 = B.from_workload(w)
    g2 = B.from_workload(w)
    got = g2.invert_eos_table(tb["axes"], tb["axis_kind"], tb["col_ids"], out=True)
    ref = tb["data"]
    den = np.maximum(np.abs(ref), np.abs(ref[..., :1]))
    assert np.max(np.abs(got - ref) / den) <= 1e-10
    g2.load_particles(w.fields)
    g1.step(5); g2.step(5)
    g1.synchronize(); g2.synchronize()
    ids = [B.R1, B.R2, B.U1, B.U2, B.S, B.NB, B.T, B.P]
    f1, f2 = g1.read_fields(ids), g2.read_fields(ids)
    for k in ids:
        d = np.max(np.abs(f1[k] - f2[k])) / max(np.max(np.abs(f1[k])), 1e-300)
        assert d <= 1e-9, (k, d)
    g1.close(); g2.close()


def test_invert_rejects_bad_arguments():
    g, _ = _ctx()
    tb = W.make_eos_table(100, 4, with_wq=False)
    axes = [a.copy() for a in tb["axes"]]
    with pytest.raises(B.CcakeError):
        g.invert_eos_table(axes, [1, 1, 1, 1], tb["col_ids"])          # axis 0 must be s itself
    with pytest.raises(B.CcakeError):
        g.invert_eos_table(axes, tb["axis_kind"], [0, 1, 2, 99])       # unknown column id
    g.close()
