"""NEXT-3 (part) of SURVEY.md §8(f): the source smearing of PAPER.md Eq. 35 (ccake_smear_sources) against the oracle
(oracle_smear_sources), element by element on seeded partons."""
import numpy as np
import pytest

import oracle as O
from paper_2511_22852_b200 import binding as B
from paper_2511_22852_b200 import workloads as W

from gpu_common import make_pair

pytestmark = pytest.mark.gpu


def _partons(rng, npart, D, extent, x0, dx0):
    r = np.zeros((3, npart))
    r[:D] = rng.uniform(-extent, extent, (D, npart))
    p = rng.normal(0.0, 1.0, (4, npart))
    p[0] = np.abs(p[0]) + np.sqrt((p[1:] ** 2).sum(axis=0))
    t = x0 + dx0 * rng.uniform(-2.0, 1.0, npart)            # a third inside the window (x0 - dx0, x0]
    t[:4] = [x0, x0 - dx0, np.nextafter(x0 - dx0, 1e9), np.nextafter(x0, 1e9)]      # the window's edges
    return p, r, t


@pytest.mark.parametrize("name,steps", [("C1", 0), ("C1h", 3), ("C4_small", 2), ("C3_small", 2)])
def test_source_smearing_matches_oracle(name, steps):
    """j^mu per particle at the loaded state or after a few steps (moved particles, advanced x0), 1,500 partons
    (a ragged number of tiles), h_source = 1.4 fm: 1e-12 of the field norm (sums of ~500 signed terms)."""
    from test_gpu_parity import WORKLOADS
    w = WORKLOADS[name]()
    g, o = make_pair(w)
    if steps:
        g.step(steps); g.synchronize(); o.step(steps)
    D = w.params["dim"]
    x0 = w.params["x0_start"] + steps * w.params["dx0"]
    rng = np.random.default_rng(35 + steps)
    ext = float(np.max(np.abs(w.fields[B.R1]))) + 1.0
    p, r, t = _partons(rng, 1500, D, ext, x0, w.params["dx0"])
    jg = g.smear_sources(p, r, t, 1.4, 0.62)
    jo = o.smear_sources(p, r, t, 1.4, 0.62)
    assert np.all(np.isfinite(jg))
    for m in range(4):
        assert np.max(np.abs(jg[m] - jo[m])) <= 1e-12 * np.max(np.abs(jo[m])), m
    assert np.max(np.abs(jo[0])) > 0
    # no parton in the window, and no parton at all
    z = g.smear_sources(p, r, np.full(1500, x0 + 1.0), 1.4, 0.62)
    assert np.all(z == 0.0)
    z = g.smear_sources(np.zeros((4, 0)), np.zeros((3, 0)), np.zeros(0), 1.4, 0.62)
    assert np.all(z == 0.0)
    g.close()


@pytest.mark.parametrize("name", ["C1", "C1h", "C4_small", "C3_small", "cloud3_hyp_dnmr_rk4"])
def test_sources_in_the_equations_of_motion(name):
    """Rest of NEXT-3, Eq. 38 / 42-44 / 96: 1,500 partons per step smeared onto the particles (Eq. 35), fed
    back as I^mu together with seeded charge sources I_q, for 4 steps (dynamical initialisation: new partons every
    step).  Rates at the first step 1e-10 of the field norm, every evolved field 1e-8 after the run; switching the
    sources off restores the source-free rates bit by bit."""
    from test_gpu_parity import WORKLOADS
    from gpu_common import TOL_GRAD, TOL_RUN, assert_fields, state_ids
    w = WORKLOADS[name]()
    g, o = make_pair(w)
    D = w.params["dim"]
    dx0 = w.params["dx0"]
    ext = float(np.max(np.abs(w.fields[B.R1]))) * 0.6
    rate_ids = [B.RATE + k for k in state_ids(w.params)]
    free = g.read_fields(rate_ids)
    rng = np.random.default_rng(96)
    scale = float(np.mean(w.fields[B.S])) * 0.02
    for step in range(4):
        x0 = w.params["x0_start"] + step * dx0
        p, r, t = _partons(rng, 1500, D, ext, x0, dx0)
        jg = g.smear_sources(p * scale, r, t, 1.4, 0.62)
        jo = o.smear_sources(p * scale, r, t, 1.4, 0.62)
        iq = 0.01 * scale * rng.normal(0.0, 1.0, (3, w.n)) * np.abs(jo[0]) / max(np.abs(jo[0]).max(), 1e-300)
        g.set_sources(jg, iq)
        o.set_sources(jo, iq)
        if step == 0:
            assert_fields(g, o, rate_ids, TOL_GRAD, name + " rates with sources")
            with_src = g.read_fields(rate_ids)
            assert any(np.max(np.abs(with_src[k] - free[k])) > 0 for k in rate_ids)
        g.step(1)
        o.step(1)
    g.synchronize(strict=False)
    assert_fields(g, o, state_ids(w.params), TOL_RUN, name + " state after 4 steps with sources")
    g.close()
    # off again: identical to a context that never had sources
    g1 = B.from_workload(w)
    g1.set_sources(np.ones((4, w.n)), None)
    g1.set_sources(None, None)
    again = g1.read_fields(rate_ids)
    for k in rate_ids:
        assert np.array_equal(again[k], free[k])
    g1.close()
