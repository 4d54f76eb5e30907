"""Edge cases of the C ABI on the GPU: degenerate inputs, ragged sizes, error codes (-m gpu)."""
import ctypes as C

import numpy as np
import pytest

import oracle as O
from paper_2511_22852_b200 import binding as B
from paper_2511_22852_b200 import workloads as W

from gpu_common import TOL_GRAD, TOL_RUN, TOL_SUM, assert_cells_equal, assert_fields, assert_neighbours_equal, make_pair, state_ids

pytestmark = pytest.mark.gpu


def _ideal(n_fields, D=2, coords=0, **kw):
    p = W.base_params(dim=D, coords=coords, eom=0, eos_kind=0, h=0.3, x0_start=1.0, dx0=0.02)
    p.update(kw)
    return W.Workload("edge", p, n_fields, None, 3, {})


def test_single_particle():
    """N = 1: sigma* = m W(0); no neighbours; zero force."""
    w = _ideal({B.R1: np.array([0.3]), B.R2: np.array([-0.2]), B.S: np.array([2.0])})
    g, o = make_pair(w)
    assert_neighbours_equal(g, o) == 0
    assert_fields(g, o, [B.SIGMA_STAR, B.S_STAR, B.T, B.P], TOL_SUM, "single")
    g.step(3)
    o.step(3)
    assert_fields(g, o, state_ids(w.params), TOL_RUN, "single after run")


def test_two_particles_apart_and_coincident():
    """Two particles farther than 2h do not interact; two coincident particles see W(0) and a zero gradient."""
    for sep in (5.0, 0.0, 0.59999, 0.6, 0.60001):
        w = _ideal({B.R1: np.array([0.0, sep]), B.R2: np.array([0.0, 0.0]), B.S: np.array([2.0, 3.0])})
        g, o = make_pair(w)
        assert_cells_equal(g, o)
        assert_neighbours_equal(g, o)
        assert_fields(g, o, [B.SIGMA_STAR, B.S_STAR, B.T, B.P], TOL_SUM, f"pair sep={sep}")
        assert_fields(g, o, [B.RATE + B.U1, B.RATE + B.U2, B.DIVV], TOL_GRAD, f"pair rates sep={sep}")
        g.close()


@pytest.mark.parametrize("n", [31, 32, 33, 255, 257, 4097])
def test_ragged_sizes(n):
    """Sizes around the warp, block and sort-tile boundaries (3-D random cloud, closed-form EoS)."""
    rng = np.random.default_rng(n)
    side = max(1.0, (n / 40.0) ** (1 / 3))
    f = {B.R1: rng.uniform(0, side, n), B.R2: rng.uniform(0, side, n), B.R3: rng.uniform(0, side, n),
         B.U1: rng.normal(0, 0.2, n), B.U2: rng.normal(0, 0.2, n), B.U3: rng.normal(0, 0.2, n),
         B.S: rng.uniform(0.5, 1.5, n), B.NB: rng.uniform(-0.01, 0.01, n), B.MASS: rng.uniform(0.5, 1.5, n)}
    w = _ideal(f, D=3, coords=1)
    g, o = make_pair(w)
    assert_cells_equal(g, o)
    assert_neighbours_equal(g, o)
    assert_fields(g, o, [B.SIGMA_STAR, B.S_STAR, B.RHOSTAR_B], TOL_SUM, "ragged sums")
    g.step(2)
    o.step(2)
    assert_fields(g, o, state_ids(w.params), TOL_RUN, "ragged after run")
    g.close()


def test_all_particles_in_one_cell_and_on_a_line():
    """Degenerate geometry: every particle inside one traversal cell; zero extent along y."""
    rng = np.random.default_rng(5)
    n = 300
    w = _ideal({B.R1: rng.uniform(0, 0.5, n), B.R2: np.zeros(n), B.S: rng.uniform(0.5, 1.5, n)})
    g, o = make_pair(w)
    assert_cells_equal(g, o)
    assert_neighbours_equal(g, o)
    assert_fields(g, o, [B.SIGMA_STAR, B.S_STAR], TOL_SUM, "one cell")
    assert_fields(g, o, [B.RATE + B.U1, B.RATE + B.U2], TOL_GRAD, "one cell rates")
    g.close()


def test_sparse_wide_domain_coarsens_grid():
    """A few particles spread over a huge box: the traversal grid is coarsened to fit the sort key, neighbour
    sets stay exact."""
    rng = np.random.default_rng(6)
    n = 500
    x = np.concatenate([rng.uniform(0, 3.0, n - 2), [-4.0e4, 5.0e4]])
    y = np.concatenate([rng.uniform(0, 3.0, n - 2), [3.0e4, -2.0e4]])
    w = _ideal({B.R1: x, B.R2: y, B.S: rng.uniform(0.5, 1.5, n)})
    w.params["neighbour_mode"] = 1      # the oracle's O(N^2) definition: its own cell list would need 1e10 cells here
    g, o = make_pair(w)
    assert_neighbours_equal(g, o)
    assert_fields(g, o, [B.SIGMA_STAR, B.S_STAR], TOL_SUM, "sparse")
    g.close()


def test_out_of_table_is_counted_and_clamped():
    """Particles outside the EoS table: coordinates clamped, ERANGE reported, state still readable, and the
    count equals the oracle's."""
    tb = W.make_eos_table(100, 6, with_wq=False)
    w = W.config_c2(n=30, dx=0.1, nsteps=2, table=tb)
    f = dict(w.fields)
    f[B.NB] = f[B.NB] * 30.0          # rho_B / s far beyond the table's +-0.05
    w = W.Workload("oob", w.params, f, tb, 2, {})
    g, o = make_pair(w)
    tg, to = g.conserved_totals(), o.conserved_totals()
    assert tg[11] == to[11] > 0
    assert_fields(g, o, [B.T, B.P, B.MU_B], TOL_SUM, "clamped thermo")
    g.step(1)
    assert g.synchronize(strict=False) == B.ERANGE
    assert np.all(np.isfinite(g.read_fields([B.U1])[B.U1]))
    g.close()


def test_error_codes():
    L = B.lib()
    bad = B.make_params(**W.base_params(dim=4))
    h = C.c_void_p()
    assert L.ccake_create(C.byref(bad), C.byref(h)) == B.EINVAL
    assert L.ccake_create(None, C.byref(h)) == B.EINVAL
    bad = B.make_params(**W.base_params(coords=1, x0_start=0.0))
    assert L.ccake_create(C.byref(bad), C.byref(h)) == B.EINVAL
    bad = B.make_params(**W.base_params(), device=99)
    assert L.ccake_create(C.byref(bad), C.byref(h)) == B.EINVAL
    g = B.Ccake(**W.base_params(eos_kind=1))
    assert L.ccake_step(g._h, 1) == B.ESTATE
    out = (C.c_double * 16)()
    assert L.ccake_conserved_totals(g._h, out) == B.ESTATE
    assert b"before load" in L.ccake_last_error(g._h)
    with pytest.raises(B.CcakeError):
        g.load_particles({99: np.zeros(4)})
    g.load_particles({B.R1: np.arange(4.0), B.R2: np.zeros(4), B.S: np.ones(4)})
    assert L.ccake_step(g._h, 1) == B.ESTATE          # table EoS selected but no table loaded
    assert L.ccake_step(g._h, -1) == B.EINVAL
    tb = W.make_eos_table(20, 4, with_wq=False)
    with pytest.raises(B.CcakeError):
        g.load_eos_table([tb["axes"][0][::-1].copy()] + tb["axes"][1:], tb["axis_kind"], tb["col_ids"], tb["data"])
    with pytest.raises(B.CcakeError):
        g.load_eos_table(tb["axes"], tb["axis_kind"], tb["col_ids"][:5], tb["data"][..., :5].copy())
    g.load_eos_table(tb["axes"], tb["axis_kind"], tb["col_ids"], tb["data"])
    assert L.ccake_step(g._h, 0) == B.OK
    ids = (C.c_int32 * 1)(B.R1)
    buf = np.zeros(2)
    ptrs = (C.c_void_p * 1)(buf.ctypes.data)
    assert L.ccake_read_fields(g._h, 1, ids, ptrs, 2, B.HOST) == B.EINVAL     # capacity < n
    g.close()


def test_reload_resets_time_and_state():
    w = W.config_c1(n=20)
    g, o = make_pair(w)
    g.step(3)
    g.load_particles(w.fields)
    assert g.conserved_totals()[0] == w.params["x0_start"]
    g.step(2)
    o.step(2)
    assert_fields(g, o, state_ids(w.params), TOL_RUN, "after reload")
    g.close()
