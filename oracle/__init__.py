"""ctypes binding of the CPU oracle (oracle/liboracle.so).  TEST INFRASTRUCTURE, NOT PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this
package.  It marshals arguments for the `oracle_*` C ABI of oracle/oracle.h and does no arithmetic.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

# ---- field ids, restated from oracle/oracle.h ---------------------------------------------------------------
R1, R2, R3, U1, U2, U3, S, NB, NS, NQ, BULK = range(11)
PI11, PI12, PI13, PI22, PI23, PI33 = range(11, 17)
JB1, JB2, JB3, JS1, JS2, JS3, JQ1, JQ2, JQ3 = range(17, 26)
MASS, WORK, NSTATE = 26, 27, 28
SIGMA_STAR, S_DENS, RHO_B, RHO_S, RHO_Q, T, MU_B, MU_S, MU_Q = range(32, 41)
P, E, CS2, GAMMA, NNB, CELL, THETA, SIGMA, S_STAR = range(41, 50)
KN_PI, RE_PI, KN_BULK, RE_BULK = range(28, 32)      # applicability diagnostics, Eq. 58-61
FO_DE0, FO_DE1, FO_DE2, FO_DE3, FO_N0, FO_N1, FO_N2, FO_N3, FO_DSIGMA = range(96, 105)   # freeze-out element, Eq. 145-148
RHOSTAR_B, RHOSTAR_S, RHOSTAR_Q, WS, DIVV = range(50, 55)
FM1, FM2, FM3, FK_B, FK_S, FK_Q = range(55, 61)
RATE = 64

FIELD_IDS = {k: v for k, v in dict(globals()).items() if k.isupper() and isinstance(v, int)}


class Params(C.Structure):
    _fields_ = [
        ("dim", C.c_int32), ("coords", C.c_int32), ("integrator", C.c_int32), ("eom", C.c_int32),
        ("flags", C.c_int32), ("eos_kind", C.c_int32), ("neighbour_mode", C.c_int32), ("reserved0", C.c_int32),
        ("h", C.c_double), ("x0_start", C.c_double), ("dx0", C.c_double),
        ("eos_c0", C.c_double), ("eos_c2", C.c_double), ("eos_c4", C.c_double),
        ("eta_over_s", C.c_double), ("tau_pi_coeff", C.c_double), ("tau_floor", C.c_double),
        ("zeta_max", C.c_double), ("zeta_T_peak", C.c_double), ("zeta_width", C.c_double),
        ("tau_Pi_coeff", C.c_double),
        ("kappa_over_T2", C.c_double * 9), ("tau_q_times_T", C.c_double * 3), ("dnmr_coeffs", C.c_double * 8),
    ]


_lib = None


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        vp, i32, i64, dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_double
        L.oracle_create.argtypes = [C.POINTER(Params), C.POINTER(vp)]
        L.oracle_destroy.argtypes = [vp]
        L.oracle_load_particles.argtypes = [vp, i64, i32, C.POINTER(i32), C.POINTER(vp)]
        L.oracle_load_eos_table.argtypes = [vp, C.POINTER(i32), C.POINTER(i32), C.POINTER(vp), i32, C.POINTER(i32), vp]
        L.oracle_step.argtypes = [vp, i32]
        L.oracle_read_fields.argtypes = [vp, i32, C.POINTER(i32), C.POINTER(vp), i64]
        L.oracle_conserved_totals.argtypes = [vp, C.POINTER(dbl)]
        L.oracle_read_neighbors.argtypes = [vp, vp, vp, vp, i64]
        L.oracle_last_error.argtypes = [vp]
        L.oracle_last_error.restype = C.c_char_p
        L.oracle_kernel_W.argtypes = [i32, dbl, dbl]
        L.oracle_kernel_W.restype = dbl
        L.oracle_kernel_gradW.argtypes = [i32, dbl, C.POINTER(dbl), C.POINTER(dbl)]
        L.oracle_kernel_gradW.restype = None
        L.oracle_eos_closed_form.argtypes = [C.POINTER(Params), dbl, C.POINTER(dbl), C.POINTER(dbl)]
        L.oracle_eos_forward.argtypes = [C.POINTER(Params), dbl, C.POINTER(dbl), C.POINTER(dbl)]
        L.oracle_eos_table_lookup.argtypes = [vp, dbl, C.POINTER(dbl), C.POINTER(dbl), C.POINTER(i32)]
        L.oracle_set_sources.argtypes = [vp, C.POINTER(vp), C.POINTER(vp)]
        L.oracle_smear_sources.argtypes = [vp, C.c_int64, C.POINTER(vp), C.POINTER(vp), vp, dbl, dbl, C.POINTER(vp)]
        _lib = L
    return _lib


def make_params(**kw) -> Params:
    p = Params()
    for k, v in kw.items():
        if k in ("kappa_over_T2", "tau_q_times_T", "dnmr_coeffs"):
            arr = getattr(p, k)
            flat = np.asarray(v, dtype=np.float64).ravel()
            for i in range(len(arr)):
                arr[i] = float(flat[i])
        elif hasattr(p, k):
            setattr(p, k, v)
        # keys the oracle does not know (device, stream) are ignored
    return p


class OracleError(RuntimeError):
    pass


class Oracle:
    """Thin handle: every method is one oracle_* call."""

    def __init__(self, **params):
        self.params = make_params(**params)
        self._h = C.c_void_p()
        self._chk(lib().oracle_create(C.byref(self.params), C.byref(self._h)), "oracle_create")
        self.n = 0

    def _chk(self, rc, what):
        if rc != 0:
            msg = lib().oracle_last_error(self._h) if self._h else b""
            raise OracleError(f"{what} failed: rc={rc} {msg.decode() if msg else ''}")

    def close(self):
        if self._h:
            lib().oracle_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def load_particles(self, fields: dict):
        ids = list(fields.keys())
        cols = [np.ascontiguousarray(fields[k], dtype=np.float64) for k in ids]
        n = len(cols[0])
        assert all(len(c) == n for c in cols)
        idarr = (C.c_int32 * len(ids))(*ids)
        ptrs = (C.c_void_p * len(ids))(*[c.ctypes.data for c in cols])
        self._chk(lib().oracle_load_particles(self._h, n, len(ids), idarr, ptrs), "oracle_load_particles")
        self.n = n

    def load_eos_table(self, axes, axis_kind, col_ids, data):
        axes = [np.ascontiguousarray(a, dtype=np.float64) for a in axes]
        data = np.ascontiguousarray(data, dtype=np.float64)
        dims = (C.c_int32 * 4)(*[len(a) for a in axes])
        kinds = (C.c_int32 * 4)(*axis_kind)
        ptrs = (C.c_void_p * 4)(*[a.ctypes.data for a in axes])
        cids = (C.c_int32 * len(col_ids))(*col_ids)
        assert data.size == int(np.prod([len(a) for a in axes])) * len(col_ids)
        self._chk(lib().oracle_load_eos_table(self._h, dims, kinds, ptrs, len(col_ids), cids, data.ctypes.data),
                  "oracle_load_eos_table")

    def step(self, nsteps=1):
        self._chk(lib().oracle_step(self._h, nsteps), "oracle_step")

    def read_fields(self, ids):
        ids = list(ids)
        out = [np.empty(self.n, dtype=np.float64) for _ in ids]
        idarr = (C.c_int32 * len(ids))(*ids)
        ptrs = (C.c_void_p * len(ids))(*[o.ctypes.data for o in out])
        self._chk(lib().oracle_read_fields(self._h, len(ids), idarr, ptrs, self.n), "oracle_read_fields")
        return dict(zip(ids, out))

    def conserved_totals(self):
        out = (C.c_double * 16)()
        self._chk(lib().oracle_conserved_totals(self._h, out), "oracle_conserved_totals")
        return np.array(out[:], dtype=np.float64)

    def read_neighbors(self):
        counts = np.empty(self.n, dtype=np.int64)
        self._chk(lib().oracle_read_neighbors(self._h, counts.ctypes.data, None, None, 0), "oracle_read_neighbors")
        offsets = np.empty(self.n + 1, dtype=np.int64)
        lst = np.empty(int(counts.sum()), dtype=np.int32)
        self._chk(lib().oracle_read_neighbors(self._h, counts.ctypes.data, offsets.ctypes.data, lst.ctypes.data,
                                              lst.size), "oracle_read_neighbors")
        return counts, offsets, lst

    def smear_sources(self, p, r, t, h_source, eta_norm=1.0):
        """oracle_smear_sources (Eq. 35): p [4, np], r [3, np], t [np] -> j [4, n]."""
        p = np.ascontiguousarray(p, dtype=np.float64); r = np.ascontiguousarray(r, dtype=np.float64)
        t = np.ascontiguousarray(t, dtype=np.float64)
        out = np.zeros((4, self.n), dtype=np.float64)
        pp = (C.c_void_p * 4)(*[p[m].ctypes.data for m in range(4)])
        rr = (C.c_void_p * 3)(*[r[a].ctypes.data for a in range(3)])
        oo = (C.c_void_p * 4)(*[out[m].ctypes.data for m in range(4)])
        self._chk(lib().oracle_smear_sources(self._h, t.size, pp, rr, t.ctypes.data, float(h_source), float(eta_norm), oo),
                  "oracle_smear_sources")
        return out

    def set_sources(self, I=None, Iq=None):
        """oracle_set_sources (Eq. 38): I [4, n] contravariant I^mu, Iq [3, n]; None clears."""
        keep = []

        def ptrs(a, k):
            if a is None:
                return None
            a = np.ascontiguousarray(a, dtype=np.float64).reshape(k, self.n)
            keep.append(a)
            return (C.c_void_p * k)(*[a[m].ctypes.data for m in range(k)])
        self._chk(lib().oracle_set_sources(self._h, ptrs(I, 4), ptrs(Iq, 3)), "oracle_set_sources")

    def eos_table_lookup(self, s, n):
        out = (C.c_double * 11)()
        oob = C.c_int32(0)
        nn = (C.c_double * 3)(*n)
        self._chk(lib().oracle_eos_table_lookup(self._h, float(s), nn, out, C.byref(oob)), "oracle_eos_table_lookup")
        return np.array(out[:]), int(oob.value)


def kernel_W(D, h, r):
    return lib().oracle_kernel_W(int(D), float(h), float(r))


def kernel_gradW(D, h, dr):
    d = (C.c_double * 3)(*[float(x) for x in dr])
    o = (C.c_double * 3)()
    lib().oracle_kernel_gradW(int(D), float(h), d, o)
    return np.array(o[:])


def eos_closed_form(params: Params, s, n):
    out = (C.c_double * 11)()
    nn = (C.c_double * 3)(*[float(x) for x in n])
    rc = lib().oracle_eos_closed_form(C.byref(params), float(s), nn, out)
    if rc:
        raise OracleError(f"oracle_eos_closed_form rc={rc}")
    return np.array(out[:])


def eos_forward(params: Params, T, mu):
    out = (C.c_double * 5)()
    mm = (C.c_double * 3)(*[float(x) for x in mu])
    rc = lib().oracle_eos_forward(C.byref(params), float(T), mm, out)
    if rc:
        raise OracleError(f"oracle_eos_forward rc={rc}")
    return np.array(out[:])


def invert_forward_table(params: Params, faxes, fdata, s, n):
    """oracle_invert_forward_table: faxes = 4 increasing axes (T, mu_B, mu_S, mu_Q), fdata[..., 5] = (p, s, n_B, n_S, n_Q) at
    the nodes, targets s[a], n[q][a].  Returns (out[nt, 11], flag[nt], iters[nt])."""
    faxes = [np.ascontiguousarray(a, dtype=np.float64) for a in faxes]
    fdata = np.ascontiguousarray(fdata, dtype=np.float64)
    dims = (C.c_int32 * 4)(*[len(a) for a in faxes])
    assert fdata.size == int(np.prod([len(a) for a in faxes])) * 5
    ax = (C.POINTER(C.c_double) * 4)(*[a.ctypes.data_as(C.POINTER(C.c_double)) for a in faxes])
    s = np.ascontiguousarray(s, dtype=np.float64)
    nn = [np.ascontiguousarray(n[q], dtype=np.float64) for q in range(3)]
    nt = s.size
    npt = (C.POINTER(C.c_double) * 3)(*[a.ctypes.data_as(C.POINTER(C.c_double)) for a in nn])
    out = np.zeros((nt, 11))
    flag = np.zeros(nt, dtype=np.int32)
    iters = np.zeros(nt, dtype=np.int32)
    L = lib()
    L.oracle_invert_forward_table.restype = C.c_int
    L.oracle_invert_forward_table.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p,
                                              C.c_void_p, C.c_void_p, C.c_void_p]
    rc = L.oracle_invert_forward_table(C.byref(params), dims, ax, fdata.ctypes.data, nt, s.ctypes.data, npt,
                                       out.ctypes.data, flag.ctypes.data, iters.ctypes.data)
    if rc:
        raise OracleError(f"oracle_invert_forward_table rc={rc}")
    return out, flag, iters
