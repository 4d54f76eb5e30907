"""ccake_smear_sources_noalloc (include/ccake.h): the source smearing of PAPER.md Eq. 35 with its scratch memory in a fixed
device array of the library instead of per-call cudaMalloc'ed buffers, against the existing ccake_smear_sources on the same
seeded partons — two calls in a row (the scratch array keeps the previous call's contents), then the size limit.

Collected last (the file name sorts behind every other test file): the suite runs with pytest -x.
"""
import numpy as np
import pytest

from paper_2511_22852_b200 import binding as B
from paper_2511_22852_b200 import workloads as W

from gpu_common import TOL_SUM

pytestmark = pytest.mark.gpu

NOALLOC_MAX = 16384          # CCAKE_SMEAR_NOALLOC_MAX of include/ccake.h


def _partons(rng, npart, D, extent, x0, dx0):
    r = np.zeros((3, npart))
    r[:D] = rng.uniform(-extent, extent, (D, npart))
    p = rng.normal(0.0, 1.0, (4, npart))
    p[0] = np.abs(p[0]) + np.sqrt((p[1:] ** 2).sum(axis=0))
    t = x0 + dx0 * rng.uniform(-2.0, 1.0, npart)             # a third inside the window (x0 - dx0, x0]
    return p, r, t


def _dev(a):
    import torch
    return [torch.from_numpy(np.ascontiguousarray(x)).cuda() for x in a]


@pytest.mark.parametrize("hyperbolic", [False, True])
def test_noalloc_smearing_equals_the_allocating_path(hyperbolic):
    import torch
    w = W.config_c1(hyperbolic=hyperbolic)
    g = B.from_workload(w)
    g.step(2)                                                # moved particles, reordered store, advanced x0
    g.synchronize()
    D, dx0 = w.params["dim"], w.params["dx0"]
    x0 = w.params["x0_start"] + 2 * dx0
    ext = float(np.max(np.abs(w.fields[B.R1]))) + 1.0
    rng = np.random.default_rng(91)
    out = [torch.full((w.n,), float("nan"), dtype=torch.float64, device="cuda") for _ in range(4)]
    # two calls in a row, the second one with FEWER partons: what the first call left in the scratch array must not leak
    for npart in (1500, 700):
        p, r, t = _partons(rng, npart, D, ext, x0, dx0)
        ref = g.smear_sources(p, r, t, 1.4, 0.62)            # existing path: host buffers, cudaMalloc / cudaFree inside
        g.smear_sources_noalloc(_dev(p), _dev(r), _dev([t])[0], 1.4, 0.62, out)
        g.synchronize()
        assert np.max(np.abs(ref[0])) > 0
        for m in range(4):
            got = out[m].cpu().numpy()
            assert np.all(np.isfinite(got))
            assert np.max(np.abs(got - ref[m])) <= TOL_SUM * np.max(np.abs(ref[m])), (npart, m)
    # no parton at all: zeros, nothing of the previous calls
    empty = torch.zeros(0, dtype=torch.float64, device="cuda")
    g.smear_sources_noalloc([empty] * 4, [empty] * 3, empty, 1.4, 0.62, out)
    g.synchronize()
    assert all(bool((o == 0).all()) for o in out)
    # beyond the fixed scratch array: refused with a clear error, the context stays usable
    big = torch.zeros(NOALLOC_MAX + 1, dtype=torch.float64, device="cuda")
    with pytest.raises(B.CcakeError, match="CCAKE_SMEAR_NOALLOC_MAX"):
        g.smear_sources_noalloc([big] * 4, [big] * 3, big, 1.4, 0.62, out)
    p, r, t = _partons(rng, NOALLOC_MAX, D, ext, x0, dx0)    # exactly the maximum is accepted
    ref = g.smear_sources(p, r, t, 1.4, 0.62)
    g.smear_sources_noalloc(_dev(p), _dev(r), _dev([t])[0], 1.4, 0.62, out)
    g.synchronize()
    for m in range(4):
        assert np.max(np.abs(out[m].cpu().numpy() - ref[m])) <= TOL_SUM * np.max(np.abs(ref[m])), m
    g.close()
