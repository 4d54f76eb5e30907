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
