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


# ------------------------------------------------------------- rest of NEXT-1: a TABULATED forward EoS (reading 21) ----
def _fwd_compare(ft, tb, n_sample, seed):
    g, P = _ctx()
    got, flags, nb = g.invert_forward_table(ft["axes"], ft["data"], tb["axes"], tb["axis_kind"], tb["col_ids"], out=True)
    assert got.shape == tb["data"].shape and np.all(np.isfinite(got)) and nb == int(flags.sum())
    ax = tb["axes"]
    rng = np.random.default_rng(seed)
    idx = np.stack([rng.integers(0, len(a), n_sample) for a in ax], axis=1)
    line = np.arange(len(ax[0]))
    idx = np.concatenate([idx, np.stack([line, 0 * line, 0 * line, 0 * line], axis=1),
                          np.stack([line, 0 * line + len(ax[1]) - 1, 0 * line, 0 * line + len(ax[3]) - 1], axis=1)])
    s = ax[0][idx[:, 0]]
    n = [ax[1 + q][idx[:, 1 + q]] * s for q in range(3)]
    ref, rflag, _ = O.invert_forward_table(P, ft["axes"], ft["data"], s, n)
    val = got[idx[:, 0], idx[:, 1], idx[:, 2], idx[:, 3]]
    gflag = flags[idx[:, 0], idx[:, 1], idx[:, 2], idx[:, 3]]
    assert np.array_equal(gflag, rflag), "the two sides disagree on which nodes fall to the backup EoS"
    # scale per column: T for T, mu, dw/ds, dw/dn; the column itself for p, e; 1 for c_s^2
    T = np.abs(ref[:, 0])
    scale = np.stack([T, T, T, T, np.abs(ref[:, 4]), np.ones_like(T), np.abs(ref[:, 6]), T, T, T, T], axis=1)
    err = np.abs(val - ref) / scale
    assert np.max(err[rflag == 0]) <= 1e-10, (np.max(err[rflag == 0], axis=0))
    if np.any(rflag == 1):
        assert np.max(err[rflag == 1]) <= 1e-12
    g.close()
    return rflag, nb, flags.size


def test_forward_table_inversion_matches_oracle_node_by_node():
    """BASELINE.json configs[1]'s shapes: forward table 100 x 32^3 on (T, mu), target grid 100 x 12^3 on (s, n_q / s).
    Sampled nodes and two corner lines against oracle_invert_forward_table: identical flags, 1e-10 at converged nodes."""
    ft = W.make_forward_table(100, 32)
    tb = W.make_eos_table(100, 12, with_wq=True)
    rflag, nb, _ = _fwd_compare(ft, tb, 1500, 22852)
    assert nb == 0 and not np.any(rflag)


def test_forward_table_inversion_backup_eos_where_the_table_ends():
    """A forward table that starts at T = 0.02 fm^-1 and ends at 1 fm^-1 cannot reach the coldest and hottest target
    decades: those nodes take the backup EoS (closed-form conformal, PAPER.md :572) on both sides, the rest converge."""
    ft = W.make_forward_table(40, 16, T_lo=0.02, T_hi=1.0, mu_lo=1e-3, mu_hi=1.2)
    tb = W.make_eos_table(100, 6, with_wq=True)
    rflag, nb, total = _fwd_compare(ft, tb, 1500, 7)
    assert 0 < nb < total and np.any(rflag == 1) and np.any(rflag == 0)


def test_run_on_the_numerically_inverted_table_matches_the_oracle_on_the_same_table():
    """The device-inverted table drives the path: the oracle, loaded with that very table, gives the same fields."""
    ft = W.make_forward_table(60, 16)
    tb = W.make_eos_table(100, 8, with_wq=False)
    w = W.config_c2(n=60, dx=0.1, nsteps=5, table=tb)
    g = B.from_workload(w)
    got, flags, nb = g.invert_forward_table(ft["axes"], ft["data"], tb["axes"], tb["axis_kind"], tb["col_ids"], out=True)
    g.load_particles(w.fields)
    o = O.Oracle(**w.params)
    o.load_eos_table(tb["axes"], tb["axis_kind"], tb["col_ids"], got)
    o.load_particles(w.fields)
    g.step(5); g.synchronize(); o.step(5)
    ids = [B.R1, B.R2, B.U1, B.U2, B.S, B.NB, B.T, B.P, B.E]
    fg, fo = g.read_fields(ids), o.read_fields(ids)
    for k in ids:
        d = np.max(np.abs(fg[k] - fo[k])) / max(np.max(np.abs(fo[k])), 1e-300)
        assert d <= 1e-8, (k, d)
    g.close()


def test_forward_inversion_rejects_bad_arguments():
    g, _ = _ctx()
    ft = W.make_forward_table(8, 4)
    tb = W.make_eos_table(100, 4, with_wq=False)
    bad = [a.copy() for a in ft["axes"]]
    bad[1] = bad[1][::-1].copy()
    with pytest.raises(B.CcakeError):
        g.invert_forward_table(bad, ft["data"], tb["axes"], tb["axis_kind"], tb["col_ids"])     # axis not increasing
    with pytest.raises(B.CcakeError):
        g.invert_forward_table(ft["axes"], ft["data"], tb["axes"], [1, 1, 1, 1], tb["col_ids"])  # axis 0 must be s
    g.close()
