"""Parity where bench.py runs (-m gpu): BASELINE.json's configs at full size in the launch configuration bench.py
times, checked on samples the oracle can afford (one whole event tile: the tiles are independent events, so the oracle
run on that tile's particles — the very same coordinates and fields, sliced from the full input — is the exact
expectation).  north_star: neighbour sets bit-exact (count plus order-free 64-bit hash of the set the PAIR KERNEL used),
smoothed densities 1e-11 per substep, fields 1e-8 after 20 RK steps.  Also: the same with a seeded non-equilibrium
start (every dissipative coupling non-trivial), and the paths of the pair kernel that a production run takes only when a
block's neighbourhood outgrows its candidate list or when device memory is short (forced by the test knobs of
include/ccake.h)."""
import os

import numpy as np
import pytest

import oracle as O
from paper_2511_22852_b200 import binding as B
from paper_2511_22852_b200 import workloads as W

from gpu_common import (POSITIVE, TOL_GRAD, TOL_RUN, TOL_SUM, assert_cells_equal, assert_fields,
                        assert_neighbours_equal, derived_ids, gradient_ids, make_pair, norm_rel, state_ids)

pytestmark = pytest.mark.gpu

_TABLES = {}


def table(ns, nq):
    if (ns, nq) not in _TABLES:
        _TABLES[(ns, nq)] = W.make_eos_table(ns, nq, with_wq=True)
    return _TABLES[(ns, nq)]


def _mix64(z):
    z = z.astype(np.uint64)
    with np.errstate(over="ignore"):
        z = z + np.uint64(0x9E3779B97F4A7C15)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
    return z ^ (z >> np.uint64(31))


def _oracle_hash(o, n, offset):
    """sum_b mix64(global original id of b + 1) over the oracle's neighbour lists of one tile (ids local to the tile)."""
    cnt, off, lst = o.read_neighbors()
    mix = _mix64(lst.astype(np.uint64) + np.uint64(offset + 1))
    ref = np.zeros(n, dtype=np.uint64)
    np.add.at(ref, np.repeat(np.arange(n), cnt), mix)
    return cnt, ref


def _tile_parity(w, tb, t, nsteps, hash_sets=True, check_rc=True):
    K = w.meta["tiles"]
    nt = w.n // K
    sl = slice(t * nt, (t + 1) * nt)
    g = B.from_workload(w)
    o = O.Oracle(**w.params)
    o.load_eos_table(tb["axes"], tb["axis_kind"], tb["col_ids"], tb["data"])
    o.load_particles({k: np.ascontiguousarray(v[sl]) for k, v in w.fields.items()})

    def compare(ids, tol, what, elementwise=()):
        fg, fo = g.read_fields(ids), o.read_fields(ids)
        bad = {}
        for k in ids:
            a, b = fg[k][sl], fo[k]
            assert np.all(np.isfinite(a)), (what, k)
            if k in elementwise:
                with np.errstate(divide="ignore", invalid="ignore"):
                    r = np.abs(a - b) / np.abs(b)
                r[a == b] = 0.0
                e = float(r.max())
            else:
                e = norm_rel(a, b)
            if not e <= tol:
                bad[k] = e
        assert not bad, f"{what}: beyond {tol:g}: {bad}"

    ng = g.read_fields([B.NNB])[B.NNB][sl]
    if hash_sets:
        cnt, ref = _oracle_hash(o, nt, t * nt)
        assert np.array_equal(ng, cnt.astype(np.float64)), "neighbour counts differ on the sampled tile"
        hg = g.neighbor_hash()[sl]
        assert np.array_equal(hg, ref), "neighbour sets used by the pair kernel differ from the oracle's (hash)"
    else:
        assert np.array_equal(ng, o.read_fields([O.NNB])[O.NNB])
    sums = [B.SIGMA_STAR, B.S_STAR, B.RHOSTAR_B, B.RHOSTAR_S, B.RHOSTAR_Q]
    compare(sums, TOL_SUM, "smoothing sums", elementwise=sums)
    compare([B.T, B.P, B.E, B.MU_B, B.MU_S, B.MU_Q], TOL_SUM, "thermodynamics")
    compare(gradient_ids(w.params), TOL_GRAD, "gradient sums")
    compare([B.RATE + k for k in state_ids(w.params)], TOL_GRAD, "rates")
    if nsteps:
        g.step(nsteps)
        rc = g.synchronize(strict=False)
        o.step(nsteps)
        compare(state_ids(w.params) + [B.SIGMA_STAR, B.T, B.P], TOL_RUN, f"fields after {nsteps} RK2 steps",
                elementwise=(B.SIGMA_STAR, B.T, B.P))
        if check_rc:
            assert rc == 0
    g.close()
    o.close()


def test_c4_full_size_tile_20_steps():
    """configs[3], 1,984,000 particles: event tile 7 of 10 — neighbour sets (count + hash from the pair kernel), sums,
    thermodynamics, gradient sums, rates, and every evolved field after 20 RK2 steps."""
    tb = table(100, 32)
    _tile_parity(W.config_c4(table=tb), tb, 7, 20)


def test_c3_full_size_tile_20_steps():
    """configs[2], 217,156 particles in 4 event tiles: tile 2, 20 RK2 steps."""
    tb = table(100, 32)
    _tile_parity(W.config_c3(table=tb), tb, 2, 20)


def test_c5_full_size_tile_one_step():
    """configs[4], 19,316,388 particles, 200x48^3 table: event tile 5 of 13 (1.49 M particles, ~1,700 neighbours each):
    one evaluation with the neighbour-set hash, then one full RK2 step."""
    tb = table(200, 48)
    _tile_parity(W.config_c5(table=tb), tb, 5, 1)


def test_c4_full_size_nonequilibrium_start():
    """configs[3] at full size with a seeded non-equilibrium start (u, Pi, pi^{ij}, J^i_q all non-zero on every
    particle): the DNMR couplings, the diffusion frame terms and the reconstruction of pi^{0 mu}, J^0 are non-trivial in
    the launch configuration bench.py times.  Tile 3, one evaluation and 5 RK2 steps."""
    tb = table(100, 32)
    w = W.with_dissipative_state(W.config_c4(table=tb), seed=4)
    _tile_parity(w, tb, 3, 5, check_rc=False)


def test_c3_full_size_nonequilibrium_start():
    tb = table(100, 32)
    w = W.with_dissipative_state(W.config_c3(table=tb), seed=3)
    _tile_parity(w, tb, 1, 5, check_rc=False)


# ------------------------------------------------------------------------------- paths forced by the test knobs ----
class knobs:
    def __init__(self, **kw):
        self.kw = {k: str(v) for k, v in kw.items()}

    def __enter__(self):
        self.old = {k: os.environ.get(k) for k in self.kw}
        os.environ.update(self.kw)

    def __exit__(self, *a):
        for k, v in self.old.items():
            if v is None:
                os.environ.pop(k, None)
            else:
                os.environ[k] = v


KNOBS = {
    "no_lists": dict(CCAKE_CAND_CAP=0),                         # every block lists its candidates inside the pass
    "lists_overflow": dict(CCAKE_CAND_CAP=1500),                # dense blocks overflow, sparse ones fit
    "no_mask_cache": dict(CCAKE_MASK_TILES=0),                  # the gradient pass culls for itself
    "short_mask_cache": dict(CCAKE_MASK_TILES=3),               # first tiles cached, the rest culled again
    "no_lists_no_masks": dict(CCAKE_CAND_CAP=0, CCAKE_MASK_TILES=0),
    "no_lists_short_masks": dict(CCAKE_CAND_CAP=0, CCAKE_MASK_TILES=5),
}


def _small(name):
    tb = W.make_eos_table(100, 8, with_wq=True)
    if name == "C4_small":
        return W.config_c4(K=2, n_side=21, n_eta=13, nsteps=20, n_hot=8, table=tb)
    if name == "C3_small":
        return W.config_c3(K=2, n_side=61, nsteps=20, n_hot=30, table=tb)
    if name == "C4_neq":
        return W.with_dissipative_state(W.config_c4(K=1, n_side=24, n_eta=13, nsteps=10, n_hot=8, table=tb), seed=9)
    raise KeyError(name)


@pytest.mark.parametrize("knob", list(KNOBS))
@pytest.mark.parametrize("name", ["C4_small", "C3_small", "C4_neq"])
def test_fallback_paths(name, knob):
    """In-pass candidate listing (several flushes of the block list, leftovers carried over), overflowing lists, and
    hit masks recomputed by the gradient pass: same bit-exact neighbour sets, same sums and fields as the oracle, and
    the same bits as the default path for everything that does not depend on the summation order."""
    w = _small(name)
    with knobs(**KNOBS[knob]):
        g, o = make_pair(w)
    assert_cells_equal(g, o)
    assert_neighbours_equal(g, o)
    cnt, ref = _oracle_hash(o, w.n, 0)
    assert np.array_equal(g.neighbor_hash(), ref)
    assert_fields(g, o, [B.SIGMA_STAR, B.S_STAR, B.SIGMA, B.S_DENS, B.GAMMA], TOL_SUM, name + " densities", elementwise=POSITIVE)
    assert_fields(g, o, derived_ids(w.params), TOL_SUM, name + " thermo")
    assert_fields(g, o, gradient_ids(w.params), TOL_GRAD, name + " gradient sums")
    assert_fields(g, o, [B.RATE + k for k in state_ids(w.params)], TOL_GRAD, name + " rates")
    assert_fields(g, o, [B.FO_DE1, B.FO_DE2], 1e-9, name + " freeze-out gradient (third pair pass)")
    g.step(6)
    g.synchronize(strict=False)
    o.step(6)
    assert_fields(g, o, state_ids(w.params), TOL_RUN, name + " state after 6 steps")
    g.close()
    o.close()


@pytest.mark.parametrize("knob", ["no_lists", "no_mask_cache", "lists_overflow"])
def test_fallback_paths_full_size_tile(knob):
    """One full-size C4 event tile (198,400 particles) through the forced paths."""
    tb = table(100, 32)
    w = W.config_c4(K=1, table=tb)
    with knobs(**KNOBS[knob]):
        g, o = make_pair(w)
    cnt, ref = _oracle_hash(o, w.n, 0)
    assert np.array_equal(g.read_fields([B.NNB])[B.NNB], cnt.astype(np.float64))
    assert np.array_equal(g.neighbor_hash(), ref)
    sums = [B.SIGMA_STAR, B.S_STAR, B.RHOSTAR_B, B.RHOSTAR_S, B.RHOSTAR_Q]
    assert_fields(g, o, sums, TOL_SUM, "smoothing sums", elementwise=sums)
    assert_fields(g, o, gradient_ids(w.params), TOL_GRAD, "gradient sums")
    g.step(1)
    g.synchronize()
    o.step(1)
    assert_fields(g, o, state_ids(w.params), TOL_RUN, "state after 1 step")
    g.close()
    o.close()


def test_runs_are_reproducible_on_fallback_paths():
    w = _small("C4_small")
    res = []
    for _ in range(2):
        with knobs(CCAKE_CAND_CAP=0, CCAKE_MASK_TILES=3):
            g = B.from_workload(w)
        g.step(3)
        res.append(g.read_fields(state_ids(w.params)))
        g.close()
    for k in res[0]:
        assert np.array_equal(res[0][k], res[1][k])


def test_out_of_table_is_reported_cumulatively():
    """a particle that is outside the EoS table in ANY substep since the load must make ccake_synchronize
    return ERANGE and show in totals[15]; totals[11] holds the latest evaluation only.  Table cut at s = 150 fm^-3: the
    hot centre of the Gubser profile (s = 175) starts above it and cools into the table during the run, so the latest
    count drops to zero while the cumulative one stays.  Both counts equal the oracle's."""
    full = W.make_eos_table(200, 8, with_wq=False)
    k = int(np.searchsorted(full["axes"][0], 150.0)) + 1
    assert abs(full["axes"][0][k - 1] - 150.0) < 1e-9
    tb = dict(full, axes=[full["axes"][0][:k].copy()] + full["axes"][1:], data=np.ascontiguousarray(full["data"][:k]))
    w = W.config_c2(n=40, dx=0.1, nsteps=8, table=tb)
    g, o = make_pair(w)
    tg, to = g.conserved_totals(), o.conserved_totals()
    assert tg[11] == to[11] > 0 and tg[15] == to[15] == 0
    g.step(8)
    rc = g.synchronize(strict=False)
    o.step(8)
    tg, to = g.conserved_totals(), o.conserved_totals()
    assert tg[11] == to[11] and tg[15] == to[15] > 0
    assert to[11] == 0, "the workload was meant to cool into the table during the run"
    assert rc == B.ERANGE
    g.close()
