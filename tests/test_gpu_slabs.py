"""Slab decomposition of ONE event over several contexts on one device (row f4 / SURVEY.md §8(e)): the slabs together must
reproduce the single-context run — neighbour counts bit-exact, smoothing sums 1e-11, fields 1e-8 after 20 steps — with halo
packing, ghost import, per-substep refresh, migration and the rebuild of the owned set all done by the library's kernels
(csrc/slab.cuh) and the messages handed over by sharding.SlabDriver.  The oracle is compared with the single-context run
elsewhere (test_gpu_parity.py); here it checks the decomposed run once more directly on a sample of fields."""
import numpy as np
import pytest
import torch

import oracle as O
from paper_2511_22852_b200 import binding as B
from paper_2511_22852_b200 import sharding as S
from paper_2511_22852_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _table():
    return W.make_eos_table(100, 8, with_wq=True)


def _with_flow(w, seed):
    """the event tiles start at rest; a seeded velocity field makes particles cross the cut planes within the run"""
    return W.with_dissipative_state(w, seed, amp=0.02, u_amp=0.25)


CASES = {
    "C4_eta_2slabs": (lambda: _with_flow(W.config_c4(K=1, n_side=20, n_eta=31, nsteps=20, n_hot=8, table=_table()), 3), 2, 2),
    "C4_eta_3slabs": (lambda: _with_flow(W.config_c4(K=1, n_side=16, n_eta=45, nsteps=20, n_hot=8, table=_table()), 4), 2, 3),
    "C3_x_3slabs": (lambda: _with_flow(W.config_c3(K=1, n_side=120, nsteps=20, n_hot=30, table=_table()), 5), 0, 3),
    "C1h_rk4_2slabs": (lambda: W.config_c1(hyperbolic=True, n=60, dx=0.2, nsteps=20, integrator=4), 0, 2),
}


def _make_slabs(w, axis, K, narrow=False):
    coord = w.fields[B.R1 + axis]
    planes = S.slab_planes(coord, K)
    width = S.slab_halo_width(w.params["h"], w.params["dx0"], narrow)
    slabs = {}
    cap = int(w.n)                      # every slab could hold the whole event: no capacity effects in the test
    for k in range(K):
        lo, hi = S.slab_bounds(planes, k)
        sel = np.nonzero((coord >= lo) & (coord < hi))[0]
        g = B.Ccake(**w.params)
        if w.table is not None:
            g.load_eos_table(w.table["axes"], w.table["axis_kind"], w.table["col_ids"], w.table["data"])
        g.slab_load({f: np.ascontiguousarray(v[sel]) for f, v in w.fields.items()}, sel.astype(np.uint32), cap, axis, lo, hi, width)
        slabs[k] = g
    nsub = 2 if w.params["integrator"] == 2 else 4
    drv = S.SlabDriver(slabs, K, nsub, cap, lambda r, c: torch.zeros((r, c), dtype=torch.float64, device="cuda:0"), narrow=narrow)
    return slabs, drv, planes


def _gather(slabs, ids, n_total):
    """owned particles of all slabs, scattered to global-id order"""
    out = {f: np.full(n_total, np.nan) for f in ids}
    seen = np.zeros(n_total, dtype=np.int32)
    for g in slabs.values():
        n_own = g.slab_info()[0]
        gid = g.slab_gids()[:n_own]
        vals = g.read_fields(ids)
        for f in ids:
            out[f][gid] = vals[f][:n_own]
        seen[gid] += 1
    assert np.all(seen == 1), "every particle must be owned by exactly one slab"
    return out


@pytest.mark.parametrize("name", list(CASES))
def test_slabs_reproduce_the_single_context_run(name):
    make, axis, K = CASES[name]
    w = make()
    ref = B.from_workload(w)
    slabs, drv, planes = _make_slabs(w, axis, K)
    state = B.state_field_ids(w.params)
    # --- the evaluation at the loaded state: neighbour counts bit-exact, smoothing sums 1e-11
    # (a slab evaluates its derived fields with the ghosts of the latest exchange: run the halo exchange of substep 0 first)
    drv.refresh_ghosts()
    ids0 = [B.NNB, B.SIGMA_STAR, B.S_STAR, B.RHOSTAR_B, B.T, B.P]
    a, b = _gather(slabs, ids0, w.n), ref.read_fields(ids0)
    assert np.array_equal(a[B.NNB], b[B.NNB]), "neighbour counts differ from the single-context run"
    for f in ids0[1:]:
        den = np.maximum(np.abs(b[f]), 1e-300)
        assert np.max(np.abs(a[f] - b[f]) / den) <= 1e-11, f
    drv.drop_ghosts()
    own0 = {k: set(g.slab_gids()[:g.slab_info()[0]].tolist()) for k, g in slabs.items()}
    # --- 20 RK steps
    drv.step(20)
    ref.step(20)
    ref.synchronize()
    a, b = _gather(slabs, state, w.n), ref.read_fields(state)
    for f in state:
        den = np.max(np.abs(b[f]))
        err = np.max(np.abs(a[f] - b[f])) / den if den > 0 else np.max(np.abs(a[f]))
        assert err <= 1e-8, (name, f, err)
    own1 = {k: set(g.slab_gids()[:g.slab_info()[0]].tolist()) for k, g in slabs.items()}
    if name != "C1h_rk4_2slabs":
        assert any(own0[k] != own1[k] for k in own0), "the run was meant to exercise migration"
    # every particle sits in the slab its coordinate belongs to
    pos = _gather(slabs, [B.R1 + axis], w.n)[B.R1 + axis]
    for k, g in slabs.items():
        lo, hi = S.slab_bounds(planes, k)
        gid = g.slab_gids()[:g.slab_info()[0]]
        assert np.all((pos[gid] >= lo) & (pos[gid] < hi))
    # conserved totals: the slabs' sums (owned particles, evaluated with fresh ghosts) add up to the single context's
    drv.refresh_ghosts()
    tot = sum(g.conserved_totals()[1:11] for g in slabs.values())
    tref = ref.conserved_totals()[1:11]
    # (momentum components are sums that cancel to rounding: measured against the size of the terms, not of the result)
    assert np.max(np.abs(tot - tref) / np.maximum(np.abs(tref), 1e-3 * np.max(np.abs(tref)))) <= 1e-9
    for g in slabs.values():
        assert g.conserved_totals()[13] == 0.0          # no bad solves among the owned particles
        g.close()
    ref.close()


@pytest.mark.parametrize("name", ["C4_eta_3slabs", "C3_x_3slabs", "C1h_rk4_2slabs"])
def test_narrow_halos_with_record_exchange(name):
    """Halos of one kernel support: the ghosts' own sums are incomplete, their gradient records come from their owners
    between a5 and a6 (ccake_slab_substep_part / export_records / import_records).  Same result as the single context, with
    about half the ghosts."""
    make, axis, K = CASES[name]
    w = make()
    ref = B.from_workload(w)
    slabs, drv, planes = _make_slabs(w, axis, K, narrow=True)
    wide, drv_w, _ = _make_slabs(w, axis, K, narrow=False)
    drv.refresh_ghosts(); drv_w.refresh_ghosts()
    g_narrow = sum(g.slab_info()[1] + g.slab_info()[2] for g in slabs.values())
    g_wide = sum(g.slab_info()[1] + g.slab_info()[2] for g in wide.values())
    assert 0 < g_narrow < 0.7 * g_wide
    for g in wide.values():
        g.close()
    a, b = _gather(slabs, [B.NNB, B.SIGMA_STAR], w.n), ref.read_fields([B.NNB, B.SIGMA_STAR])
    assert np.array_equal(a[B.NNB], b[B.NNB])
    assert np.max(np.abs(a[B.SIGMA_STAR] - b[B.SIGMA_STAR]) / b[B.SIGMA_STAR]) <= 1e-11
    drv.step(20)
    ref.step(20)
    ref.synchronize()
    state = B.state_field_ids(w.params)
    a, b = _gather(slabs, state, w.n), ref.read_fields(state)
    for f in state:
        den = np.max(np.abs(b[f]))
        err = np.max(np.abs(a[f] - b[f])) / den if den > 0 else np.max(np.abs(a[f]))
        assert err <= 1e-8, (name, f, err)
    for g in slabs.values():
        assert g.conserved_totals()[13] == 0.0
        g.close()
    ref.close()


def test_decomposed_run_against_the_oracle():
    """the decomposed run compared with the oracle itself (not only with the single-context GPU run)"""
    make, axis, K = CASES["C4_eta_2slabs"]
    w = make()
    slabs, drv, _ = _make_slabs(w, axis, K)
    o = O.Oracle(**w.params)
    o.load_eos_table(w.table["axes"], w.table["axis_kind"], w.table["col_ids"], w.table["data"])
    o.load_particles(w.fields)
    drv.step(3)
    o.step(3)
    state = B.state_field_ids(w.params)
    a, b = _gather(slabs, state, w.n), o.read_fields(state)
    for f in state:
        den = np.max(np.abs(b[f]))
        err = np.max(np.abs(a[f] - b[f])) / den if den > 0 else np.max(np.abs(a[f]))
        assert err <= 1e-8, (f, err)
    for g in slabs.values():
        g.close()


def test_slab_calls_are_refused_on_plain_contexts_and_steps_on_slab_contexts():
    w = W.config_c1(n=20, nsteps=1)
    g = B.from_workload(w)
    buf = torch.zeros((S.SLAB_ROWS, 64), dtype=torch.float64, device="cuda:0")
    with pytest.raises(B.CcakeError) as e:
        g.slab_export_halo(0, 0, buf)
    assert e.value.rc == B.ESTATE
    g.close()
    g = B.Ccake(**w.params)
    x = w.fields[B.R1]
    g.slab_load(w.fields, np.arange(w.n, dtype=np.uint32), w.n, 0, -S.INF, S.INF, 1.3)
    with pytest.raises(B.CcakeError) as e:
        g.step(1)
    assert e.value.rc == B.ESTATE
    g.slab_substep(0); g.slab_substep(1); g.slab_commit()        # a single slab without neighbours is the plain run
    ref = B.from_workload(w)
    ref.step(1)
    a, b = g.read_fields([B.S, B.U1]), ref.read_fields([B.S, B.U1])
    gid = g.slab_gids()
    for f in (B.S, B.U1):
        assert np.max(np.abs(a[f] - b[f][gid])) <= 1e-12 * max(np.max(np.abs(b[f])), 1e-300)
    g.close(); ref.close()


def test_slab_error_paths():
    """Message larger than the caller's buffer, ghosts beyond the capacity, imports in the wrong order, a second import without
    a commit: refused with the documented codes, and the context stays usable."""
    w = _with_flow(W.config_c4(K=1, n_side=12, n_eta=31, nsteps=2, n_hot=4, table=_table()), 9)
    slabs, drv, planes = _make_slabs(w, 2, 2)
    lo, hi = slabs[0], slabs[1]
    small = torch.zeros((S.SLAB_ROWS, 8), dtype=torch.float64, device="cuda:0")
    big = torch.zeros((S.SLAB_ROWS, w.n), dtype=torch.float64, device="cuda:0")
    with pytest.raises(B.CcakeError) as e:
        lo.slab_export_halo(1, 0, small)                      # hundreds of halo particles do not fit 8 columns
    assert e.value.rc == B.ENOMEM
    cnt = lo.slab_export_halo(1, 0, big)
    assert cnt > 8
    with pytest.raises(B.CcakeError) as e:
        lo.slab_export_halo(2, 0, big)                        # no such face
    assert e.value.rc == B.EINVAL
    hi.slab_import_ghosts(1, 0, big, cnt)                     # (the same particles, standing in for a high neighbour's message)
    with pytest.raises(B.CcakeError) as e:
        hi.slab_import_ghosts(0, 0, big, cnt)                 # low side after the high side
    assert e.value.rc == B.ESTATE
    hi.slab_commit()
    hi.slab_import_ghosts(0, 0, big, cnt)
    with pytest.raises(B.CcakeError) as e:
        hi.slab_import_ghosts(0, 0, big, cnt)                 # the ghosts of the first import are still there
    assert e.value.rc == B.ESTATE
    with pytest.raises(B.CcakeError) as e:
        hi.slab_import_ghosts(0, 1, big, cnt - 1)             # a later substep must bring the same particles
    assert e.value.rc == B.EINVAL
    hi.slab_commit()
    # a context loaded with no room for ghosts
    sel = np.nonzero(w.fields[B.R3] >= planes[0])[0]
    g = B.Ccake(**w.params)
    g.load_eos_table(w.table["axes"], w.table["axis_kind"], w.table["col_ids"], w.table["data"])
    g.slab_load({f: np.ascontiguousarray(v[sel]) for f, v in w.fields.items()}, sel.astype(np.uint32), sel.size, 2, planes[0], S.INF, 1.3)
    with pytest.raises(B.CcakeError) as e:
        g.slab_import_ghosts(0, 0, big, cnt)
    assert e.value.rc == B.ENOMEM
    g.close()
    # the pair of slabs still runs a step after all that
    drv.step(1)
    for s_ in slabs.values():
        assert s_.conserved_totals()[13] == 0.0
        s_.close()
