"""Parity of the CUDA library (through its C ABI) with the CPU oracle, element by element, on the same seeded
inputs (-m gpu).  Sizes span several sort tiles, many cells and ragged tails; see gpu_common.py for tolerances.
"""
import numpy as np
import pytest

import oracle as O
from paper_2511_22852_b200 import binding as B
from paper_2511_22852_b200 import workloads as W

from gpu_common import (POSITIVE, TOL_GRAD, TOL_RUN, TOL_SUM, assert_cells_equal, assert_fields,
                        assert_neighbours_equal, derived_ids, drift, gradient_ids, make_pair, norm_rel, state_ids)

pytestmark = pytest.mark.gpu

_TABLES = {}


def table(ns=100, nq=8, with_wq=True):
    key = (ns, nq, with_wq)
    if key not in _TABLES:
        _TABLES[key] = W.make_eos_table(ns, nq, with_wq=with_wq)
    return _TABLES[key]


def viscous_cloud(D, coords, eom, n_side, seed, eos_kind=1, integrator=2, dx0=0.01, flags=7):
    """Jittered lattice with a full random dissipative state (Pi, pi^ij, J^i_q all non-zero), unequal masses."""
    rng = np.random.default_rng(seed)
    dx = 0.15
    x1 = (np.arange(n_side) - (n_side - 1) / 2) * dx
    grids = np.meshgrid(*([x1] * D), indexing="ij")
    N = grids[0].size
    f = {}
    for k in range(D):
        f[B.R1 + k] = grids[k].ravel() + rng.uniform(-0.03, 0.03, N)
        f[B.U1 + k] = rng.normal(0, 0.3, N)
    vol = dx ** D
    f[B.S] = rng.uniform(20, 60, N) * vol
    for q in range(3):
        f[B.NB + q] = rng.uniform(-0.5, 0.5, N) * vol
    f[B.BULK] = rng.normal(0, 1.0, N) * vol
    for c in (B.PI11, B.PI12, B.PI22, B.PI33) + ((B.PI13, B.PI23) if D == 3 else ()):
        f[c] = rng.normal(0, 1.0, N) * vol
    for q in range(3):
        for k in range(D):
            f[B.JB1 + 3 * q + k] = rng.normal(0, 0.02, N) * vol
    f[B.MASS] = rng.uniform(0.8, 1.2, N)
    p = W.viscous_params(D, eom, dx0, x0=0.8)
    p.update(coords=coords, eos_kind=eos_kind, integrator=integrator, flags=flags)
    tb = table(100, 8, True) if eos_kind == 1 else None
    return W.Workload(f"cloud{D}d", p, f, tb, 3, {})


WORKLOADS = {
    "C1": lambda: W.config_c1(),
    "C1h": lambda: W.config_c1(hyperbolic=True),
    "C1h_rk4": lambda: W.config_c1(hyperbolic=True, integrator=4, nsteps=10),
    "C2_small": lambda: W.config_c2(n=70, dx=0.1, nsteps=20, table=table(100, 8, False)),
    "C3_small": lambda: W.config_c3(K=2, n_side=61, nsteps=20, n_hot=30, table=table()),
    "C4_small": lambda: W.config_c4(K=2, n_side=21, n_eta=13, nsteps=20, n_hot=8, table=table()),
    "C5_small": lambda: W.config_c5(K=1, n_side=34, n_eta=9, nsteps=20, n_hot=20, table=table()),
    "cloud2_cart_is": lambda: viscous_cloud(2, 0, 1, 37, 11),
    "cloud2_hyp_dnmr": lambda: viscous_cloud(2, 1, 2, 41, 12),
    "cloud3_hyp_is": lambda: viscous_cloud(3, 1, 1, 13, 13),
    "cloud3_hyp_dnmr_rk4": lambda: viscous_cloud(3, 1, 2, 12, 14, integrator=4),
    "cloud3_cart_closed": lambda: viscous_cloud(3, 0, 1, 11, 15, eos_kind=0),
    "cloud2_shear_only": lambda: viscous_cloud(2, 1, 1, 29, 16, flags=1),
    "cloud3_bulk_diff": lambda: viscous_cloud(3, 1, 1, 11, 17, flags=6),
}


@pytest.mark.parametrize("name", list(WORKLOADS))
def test_one_evaluation(name):
    """Steps a1-a7 at the loaded state: cell ids and neighbour sets bit-exact; smoothed densities 1e-11
    element-wise; thermodynamics 1e-11; gradient sums and rates 1e-10 of the field norm."""
    w = WORKLOADS[name]()
    g, o = make_pair(w)
    assert_cells_equal(g, o)
    npairs = assert_neighbours_equal(g, o)
    assert npairs > 0
    assert_fields(g, o, [B.SIGMA_STAR, B.S_STAR, B.SIGMA, B.S_DENS, B.GAMMA], TOL_SUM, name + " densities",
                  elementwise=POSITIVE)
    assert_fields(g, o, derived_ids(w.params), TOL_SUM, name + " thermo")
    assert_fields(g, o, gradient_ids(w.params), TOL_GRAD, name + " gradient sums")
    assert_fields(g, o, [B.RATE + k for k in state_ids(w.params)], TOL_GRAD, name + " rates")
    tg, to = g.conserved_totals(), o.conserved_totals()
    assert tg[14] == to[14] == npairs
    assert tg[11] == to[11]
    for k in (1, 5, 9):
        assert abs(tg[k] - to[k]) <= 1e-11 * abs(to[k])
    for k in (2, 3, 4, 6, 7, 8, 10, 12):
        assert abs(tg[k] - to[k]) <= 1e-10 * max(abs(to[k]), np.abs(to[1:10]).max() * 1e-3)
    g.close()
    o.close()


@pytest.mark.parametrize("name", list(WORKLOADS))
def test_fields_after_run(name):
    """k RK steps: every evolved field within 1e-8 (norm-wise; positive derived fields element-wise); conserved
    totals drift no more than the oracle's."""
    w = WORKLOADS[name]()
    g, o = make_pair(w)
    t0g, t0o = g.conserved_totals(), o.conserved_totals()
    nsteps = min(w.nsteps, 20)
    g.step(nsteps)
    rc = g.synchronize(strict=False)
    o.step(nsteps)
    assert_fields(g, o, state_ids(w.params), TOL_RUN, name + " state after run")
    assert_fields(g, o, [B.SIGMA_STAR, B.S_DENS, B.T, B.P], TOL_RUN, name + " derived after run", elementwise=POSITIVE)
    t1g, t1o = g.conserved_totals(), o.conserved_totals()
    assert t1g[0] == pytest.approx(t1o[0], abs=1e-12)
    assert (rc == B.ERANGE) == (t1o[15] > 0 or t1o[11] > 0), (rc, t1o[11], t1o[15])
    assert t1g[15] == t1o[15] and t1g[11] == t1o[11]
    dg, do = drift(t0g, t1g), drift(t0o, t1o)
    scale = np.abs(t0o[1:10]).max()
    for k in dg:
        assert dg[k] <= do[k] * (1 + 1e-6) + 1e-12 * (scale if k in ("P", "N") else 1.0), (k, dg, do)
    g.close()
    o.close()


@pytest.mark.parametrize("name", ["C1", "C3_small", "C4_small"])
def test_neighbours_on_evolved_state(name):
    """Bit-exact neighbour sets and cell ids on irregular positions: the oracle's evolved state is loaded into
    a fresh CUDA context, so both sides see the same bits."""
    w = WORKLOADS[name]()
    o = O.Oracle(**w.params)
    if w.table is not None:
        o.load_eos_table(w.table["axes"], w.table["axis_kind"], w.table["col_ids"], w.table["data"])
    o.load_particles(w.fields)
    o.step(5)
    ids = [k for k in state_ids(w.params) if k != B.WORK]
    st = o.read_fields(ids)
    w2 = W.Workload(w.name, w.params, st, w.table, 1, {})
    g, o2 = make_pair(w2)
    assert_cells_equal(g, o2)
    assert_neighbours_equal(g, o2)
    h1 = g.neighbor_hash()
    cnt, off, lst = o2.read_neighbors()
    mix = _mix64(lst.astype(np.uint64) + np.uint64(1))
    ref = np.zeros(w2.n, dtype=np.uint64)
    np.add.at(ref, np.repeat(np.arange(w2.n), cnt), mix)
    assert np.array_equal(h1, ref)
    g.close()


def _mix64(z):
    z = z.astype(np.uint64)
    with np.errstate(over="ignore"):
        z = z + np.uint64(0x9E3779B97F4A7C15)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
    return z ^ (z >> np.uint64(31))


def test_device_memspace_round_trip():
    """Loading from and reading into device buffers (torch tensors) gives the same result as host buffers."""
    import torch
    w = WORKLOADS["C3_small"]()
    gh = B.from_workload(w, memspace="host")
    gd = B.from_workload(w, memspace="device")
    gh.step(3)
    gd.step(3)
    ids = state_ids(w.params)
    a = gh.read_fields(ids)
    out = [torch.empty(w.n, dtype=torch.float64, device="cuda") for _ in ids]
    gd.read_fields(ids, out=out)
    for k, t in zip(ids, out):
        assert np.array_equal(a[k], t.cpu().numpy())
    gh.close()
    gd.close()


def test_runs_are_reproducible():
    """Two runs of the same input give identical bits (fixed reduction order everywhere)."""
    w = WORKLOADS["C4_small"]()
    res = []
    for _ in range(2):
        g = B.from_workload(w)
        g.step(4)
        res.append((g.read_fields(state_ids(w.params)), g.conserved_totals()))
        g.close()
    for k in res[0][0]:
        assert np.array_equal(res[0][0][k], res[1][0][k])
    assert np.array_equal(res[0][1], res[1][1])


@pytest.mark.parametrize("name", ["C1h_rk4", "C4_small"])
def test_graph_replay_equals_direct_launches(name):
    """On a non-default stream ccake_step replays one captured CUDA graph per RK step (the time lives on the device, one
    graph per physical Y[0] buffer); on the legacy default stream it launches kernel by kernel.  Same bits — also when
    reads in between (which re-sort the store and flip the buffers), a reload and a change of sources drop or switch graphs."""
    import torch
    w = WORKLOADS[name]()
    stream = torch.cuda.Stream()
    ga = B.from_workload(w, stream=stream.cuda_stream)        # graph path
    gb = B.from_workload(w)                                   # direct path
    ids = state_ids(w.params)
    rng = np.random.default_rng(5)
    src = [1e-3 * rng.normal(size=w.n) for _ in range(4)]
    for g in (ga, gb):
        g.step(3)
        g.read_fields([B.T])                                  # refresh: reorders the store, flips Y[0] / Y[1]
        g.step(2)
        g.conserved_totals()
        g.step(1)
        g.set_sources(I=src)                                  # the captured steps were recorded without sources
        g.step(2)
        g.set_sources()
        g.step(1)
        g.synchronize()
    fa, fb = ga.read_fields(ids), gb.read_fields(ids)
    for k in ids:
        assert np.array_equal(fa[k], fb[k]), k
    assert np.array_equal(ga.conserved_totals(), gb.conserved_totals())
    assert ga.launch_count() == gb.launch_count()             # the replay books the launches it stands for
    ga.load_particles(w.fields); gb.load_particles(w.fields)  # reload: time and state reset, graphs still valid or rebuilt
    ga.step(2); gb.step(2)
    fa, fb = ga.read_fields(ids), gb.read_fields(ids)
    for k in ids:
        assert np.array_equal(fa[k], fb[k]), k
    ga.close(); gb.close()


def test_async_read_equals_blocking_read():
    """ccake_read_fields_async + wait return what ccake_read_fields returns, also with steps enqueued in between and with two
    reads in flight one after the other."""
    import torch
    w = WORKLOADS["C4_small"]()
    stream = torch.cuda.Stream()
    g = B.from_workload(w, stream=stream.cuda_stream)
    ids = state_ids(w.params) + [B.T, B.SIGMA_STAR]
    bufs = [[torch.empty(w.n, dtype=torch.float64).pin_memory() for _ in ids] for _ in range(2)]
    g.step(2)
    g.read_fields_async(ids, bufs[0])
    g.step(1)                                                # enqueued while the copies of the first read run
    g.read_fields_async(ids, bufs[1])
    g.read_fields_wait()
    ref1 = g.read_fields(ids)
    for k, b in zip(ids, bufs[1]):
        assert np.array_equal(b.numpy(), ref1[k]), k
    g2 = B.from_workload(w)
    g2.step(2)
    ref0 = g2.read_fields(ids)
    for k, b in zip(ids, bufs[0]):
        assert np.array_equal(b.numpy(), ref0[k]), k
    g.close(); g2.close()


def test_staged_load_equals_blocking_load():
    """ccake_stage_particles + ccake_load_staged install what ccake_load_particles installs: the same results bit for bit,
    with the copies of the next set in flight while the resident one is stepped and read back, with a set of another size
    (the path that reallocates), and ESTATE with nothing staged."""
    import torch
    w = WORKLOADS["C4_small"]()
    stream = torch.cuda.Stream()
    g = B.from_workload(w, stream=stream.cuda_stream)
    ids = state_ids(w.params) + [B.T, B.SIGMA_STAR]
    g.step(2)
    ref = g.read_fields(ids)
    with pytest.raises(B.CcakeError):
        g.load_staged()
    rng = np.random.default_rng(5)
    fields2 = {k: v.copy() for k, v in w.fields.items()}
    fields2[B.S] = fields2[B.S] * (1.0 + 0.05 * rng.uniform(-1.0, 1.0, w.n))        # a second, different event
    pin = [{k: torch.from_numpy(np.ascontiguousarray(v)).pin_memory() for k, v in f.items()} for f in (w.fields, fields2)]
    bufs = [[torch.empty(w.n, dtype=torch.float64).pin_memory() for _ in ids] for _ in range(3)]
    g.stage_particles(pin[0])
    for it in range(3):                                      # events 0, 1, 0: load, stage the next one, step, read back
        g.load_staged()
        if it < 2:
            g.stage_particles(pin[(it + 1) % 2])
        g.step(2)
        g.read_fields_async(ids, bufs[it])
    g.read_fields_wait()
    g.synchronize()
    g2 = B.from_workload(w)
    g2.load_particles(fields2)
    g2.step(2)
    ref2 = g2.read_fields(ids)
    for k, b0, b1, b2 in zip(ids, *bufs):
        assert np.array_equal(b0.numpy(), ref[k]), k
        assert np.array_equal(b1.numpy(), ref2[k]), k
        assert np.array_equal(b2.numpy(), ref[k]), k
    # another particle count: the staged set goes through the allocating load
    m = w.n // 2
    half = {k: torch.from_numpy(np.ascontiguousarray(v[:m])).pin_memory() for k, v in w.fields.items()}
    g.stage_particles(half)
    g.load_staged()
    g.step(1)
    g2.load_particles({k: v[:m] for k, v in w.fields.items()})
    g2.step(1)
    a, b = g.read_fields(ids), g2.read_fields(ids)
    for k in ids:
        assert a[k].shape == (m,) and np.array_equal(a[k], b[k]), k
    g.close(); g2.close()


def test_full_size_c2():
    """BASELINE.json configs[1] at full size (40,000 particles, 100x32^3x8 table), whole workload on both sides:
    one evaluation, then 20 RK2 steps."""
    w = W.config_c2(nsteps=20)
    g, o = make_pair(w)
    assert_cells_equal(g, o)
    assert_neighbours_equal(g, o)
    sums = [B.SIGMA_STAR, B.S_STAR, B.RHOSTAR_B, B.RHOSTAR_S, B.RHOSTAR_Q]
    assert_fields(g, o, sums, TOL_SUM, "smoothing sums", elementwise=sums)
    g.step(20)
    g.synchronize()
    o.step(20)
    assert_fields(g, o, state_ids(w.params) + [B.SIGMA_STAR, B.T, B.P], TOL_RUN, "fields after 20 steps",
                  elementwise=(B.SIGMA_STAR, B.T, B.P))
    g.close()


@pytest.mark.parametrize("name", ["C3_small", "C4_small", "cloud2_hyp_dnmr", "cloud3_hyp_is", "cloud3_cart_closed"])
def test_applicability_diagnostics(name):
    """NEXT-4 of SURVEY.md §8(f), Eq. 58-61 (:797-805): Knudsen and inverse Reynolds numbers of shear and
    bulk per particle, at the loaded state and after 3 RK steps — 1e-9 of the field's infinity norm (they are built
    from the velocity-gradient sums, tolerance class of gradient_ids)."""
    w = WORKLOADS[name]()
    g, o = make_pair(w)
    ids = [B.KN_PI, B.RE_PI, B.KN_BULK, B.RE_BULK]
    assert (B.KN_PI, B.RE_PI, B.KN_BULK, B.RE_BULK) == (O.KN_PI, O.RE_PI, O.KN_BULK, O.RE_BULK)
    assert_fields(g, o, ids, 1e-9, "diagnostics at the loaded state")
    g.step(3)
    g.synchronize()
    o.step(3)
    assert_fields(g, o, ids, 1e-8, "diagnostics after 3 steps")
    g.close()


@pytest.mark.parametrize("name", ["C1h", "C3_small", "C4_small", "cloud2_hyp_dnmr", "cloud3_hyp_is", "cloud3_cart_closed"])
def test_freezeout_element(name):
    """NEXT-2 of SURVEY.md §8(f), §5.10 Eq. 145-148 (:1466-1482): d_mu eps, the outward normal n_mu and
    |d sigma| per particle, at the loaded state and after 2 RK steps.  d_mu eps: 1e-9 of the field norm (a signed
    SPH sum / rates); n_mu and |d sigma| are ratios of those and are compared where the gradient is not noise
    (|d eps . d eps| above 1e-6 of its maximum): 1e-7."""
    w = WORKLOADS[name]()
    g, o = make_pair(w)
    de = [B.FO_DE0, B.FO_DE1, B.FO_DE2, B.FO_DE3]
    nn = [B.FO_N0, B.FO_N1, B.FO_N2, B.FO_N3, B.FO_DSIGMA]
    assert tuple(de + nn) == (O.FO_DE0, O.FO_DE1, O.FO_DE2, O.FO_DE3, O.FO_N0, O.FO_N1, O.FO_N2, O.FO_N3, O.FO_DSIGMA)

    def check(what, tol_de, tol_n):
        fg, fo = g.read_fields(de + nn), o.read_fields(de + nn)
        scale = max(float(np.max(np.abs(fo[k]))) for k in de)
        for k in de:
            assert np.all(np.isfinite(fg[k]))
            assert np.max(np.abs(fg[k] - fo[k])) <= tol_de * scale, (what, k)
        G3 = 1.0
        inv = np.abs(fo[B.FO_DE0] ** 2 - fo[B.FO_DE1] ** 2 - fo[B.FO_DE2] ** 2 - fo[B.FO_DE3] ** 2 / G3)
        ok = inv > 1e-6 * inv.max()
        assert ok.sum() >= 0.05 * ok.size
        for k in nn:
            den = np.maximum(np.maximum(np.abs(fo[k][ok]), 1e-3 * np.max(np.abs(fo[k][ok]))), 1e-300)
            assert np.max(np.abs(fg[k][ok] - fo[k][ok]) / den) <= tol_n, (what, k)

    check("loaded state", 1e-9, 1e-7)
    g.step(2)
    g.synchronize()
    o.step(2)
    check("after 2 steps", 1e-8, 1e-6)
    g.close()
