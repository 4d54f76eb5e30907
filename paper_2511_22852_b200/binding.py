"""Thin ctypes binding of libccake.so (include/ccake.h).  Argument marshalling only: every step of the hot path
runs in the CUDA kernels of the library.  The library is loaded on first use; when it is missing or cannot be
loaded the binding raises — there is no CPU fallback.

Names follow the C ABI: Ccake.load_particles -> ccake_load_particles, etc.  Inputs may be numpy arrays (host) or
torch CUDA tensors (device, passed as data_ptr()).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libccake.so")

# ---- field ids, restated from include/ccake.h ---------------------------------------------------------------
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
HOST, DEVICE = 0, 1
OK, EINVAL, ENOMEM, ECUDA, ESTATE, ERANGE = 0, -1, -2, -3, -4, -5

EXPORTS = ["ccake_create", "ccake_destroy", "ccake_load_particles", "ccake_load_eos_table", "ccake_invert_eos_table", "ccake_invert_forward_table", "ccake_smear_sources", "ccake_smear_sources_noalloc",
           "ccake_set_sources",
           "ccake_slab_load", "ccake_slab_export_halo", "ccake_slab_import_ghosts", "ccake_slab_substep", "ccake_slab_substep_part", "ccake_slab_export_records", "ccake_slab_import_records",
           "ccake_slab_export_migrants", "ccake_slab_import_migrants", "ccake_slab_commit", "ccake_slab_info", "ccake_slab_gids",
           "ccake_step",
           "ccake_synchronize", "ccake_read_fields", "ccake_read_fields_async", "ccake_read_fields_wait", "ccake_stage_particles", "ccake_load_staged", "ccake_conserved_totals", "ccake_read_neighbors",
           "ccake_neighbor_hash", "ccake_kernel_times", "ccake_enable_timing", "ccake_launch_count",
           "ccake_measure_fp64_peak", "ccake_last_error"]


class Params(C.Structure):
    _fields_ = [
        ("dim", C.c_int32), ("coords", C.c_int32), ("integrator", C.c_int32), ("eom", C.c_int32),
        ("flags", C.c_int32), ("eos_kind", C.c_int32), ("device", C.c_int32), ("reserved0", C.c_int32),
        ("stream", C.c_void_p),
        ("h", C.c_double), ("x0_start", C.c_double), ("dx0", C.c_double),
        ("eos_c0", C.c_double), ("eos_c2", C.c_double), ("eos_c4", C.c_double),
        ("eta_over_s", C.c_double), ("tau_pi_coeff", C.c_double), ("tau_floor", C.c_double),
        ("zeta_max", C.c_double), ("zeta_T_peak", C.c_double), ("zeta_width", C.c_double),
        ("tau_Pi_coeff", C.c_double),
        ("kappa_over_T2", C.c_double * 9), ("tau_q_times_T", C.c_double * 3), ("dnmr_coeffs", C.c_double * 8),
    ]


class CcakeError(RuntimeError):
    def __init__(self, what, rc, msg=""):
        super().__init__(f"{what} failed: rc={rc} {msg}")
        self.rc = rc


_lib = None


def lib():
    """Load libccake.so; raise loudly when the CUDA extension is missing (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} not found: build it with `python -m paper_2511_22852_b200.build` "
                              "(nvcc, sm_100a).  There is no CPU fallback.")
        L = C.CDLL(LIB_PATH)
        vp, i32, i64 = C.c_void_p, C.c_int32, C.c_int64
        L.ccake_create.argtypes = [C.POINTER(Params), C.POINTER(vp)]
        L.ccake_destroy.argtypes = [vp]
        L.ccake_load_particles.argtypes = [vp, i64, i32, C.POINTER(i32), C.POINTER(vp), i32]
        L.ccake_load_eos_table.argtypes = [vp, C.POINTER(i32), C.POINTER(i32), C.POINTER(vp), i32, C.POINTER(i32), vp, i32]
        L.ccake_invert_eos_table.argtypes = [vp, C.POINTER(i32), C.POINTER(i32), C.POINTER(vp), i32, C.POINTER(i32), vp, i32]
        L.ccake_invert_forward_table.argtypes = [vp, C.POINTER(i32), C.POINTER(vp), vp, C.POINTER(i32), C.POINTER(i32), C.POINTER(vp), i32,
                                                 C.POINTER(i32), vp, vp, C.POINTER(i64), i32]
        L.ccake_smear_sources.argtypes = [vp, i64, C.POINTER(vp), C.POINTER(vp), vp, C.c_double, C.c_double, C.POINTER(vp), i32]
        L.ccake_smear_sources_noalloc.argtypes = [vp, i64, C.POINTER(vp), C.POINTER(vp), vp, C.c_double, C.c_double, C.POINTER(vp)]
        L.ccake_set_sources.argtypes = [vp, C.POINTER(vp), C.POINTER(vp), i32]
        L.ccake_slab_load.argtypes = [vp, i64, i64, i32, C.POINTER(i32), C.POINTER(vp), vp, i32, C.c_double, C.c_double, C.c_double, i32]
        L.ccake_slab_export_halo.argtypes = [vp, i32, i32, vp, i64, C.POINTER(i64)]
        L.ccake_slab_import_ghosts.argtypes = [vp, i32, i32, vp, i64, i64]
        L.ccake_slab_substep.argtypes = [vp, i32]
        L.ccake_slab_substep_part.argtypes = [vp, i32, i32]
        L.ccake_slab_export_records.argtypes = [vp, i32, vp, i64, C.POINTER(i64)]
        L.ccake_slab_import_records.argtypes = [vp, i32, vp, i64, i64]
        L.ccake_slab_export_migrants.argtypes = [vp, i32, vp, i64, C.POINTER(i64)]
        L.ccake_slab_import_migrants.argtypes = [vp, i32, vp, i64, i64]
        L.ccake_slab_commit.argtypes = [vp, C.POINTER(i64)]
        L.ccake_slab_info.argtypes = [vp, C.POINTER(i64)]
        L.ccake_slab_gids.argtypes = [vp, vp, i64, i32]
        L.ccake_step.argtypes = [vp, i32]
        L.ccake_synchronize.argtypes = [vp]
        L.ccake_read_fields.argtypes = [vp, i32, C.POINTER(i32), C.POINTER(vp), i64, i32]
        L.ccake_read_fields_async.argtypes = [vp, i32, C.POINTER(i32), C.POINTER(vp), i64]
        L.ccake_read_fields_wait.argtypes = [vp]
        L.ccake_stage_particles.argtypes = [vp, i64, i32, C.POINTER(i32), C.POINTER(vp)]
        L.ccake_load_staged.argtypes = [vp]
        L.ccake_conserved_totals.argtypes = [vp, C.POINTER(C.c_double)]
        L.ccake_read_neighbors.argtypes = [vp, vp, vp, vp, i64]
        L.ccake_neighbor_hash.argtypes = [vp, vp, i64]
        L.ccake_kernel_times.argtypes = [vp, C.POINTER(C.c_double)]
        L.ccake_enable_timing.argtypes = [vp, i32]
        L.ccake_launch_count.argtypes = [vp, C.POINTER(i64)]
        L.ccake_measure_fp64_peak.argtypes = [i32, C.POINTER(C.c_double)]
        L.ccake_last_error.argtypes = [vp]
        L.ccake_last_error.restype = C.c_char_p
        _lib = L
    return _lib


def measure_fp64_peak(device=0) -> float:
    """ccake_measure_fp64_peak: TFLOP/s of the device's FP64 pipe (DFMA chains on every SM)."""
    out = C.c_double(0.0)
    rc = lib().ccake_measure_fp64_peak(int(device), C.byref(out))
    if rc != 0:
        raise CcakeError("ccake_measure_fp64_peak", rc, "")
    return float(out.value)


def make_params(**kw) -> Params:
    p = Params()
    for k, v in kw.items():
        if k in ("kappa_over_T2", "tau_q_times_T", "dnmr_coeffs"):
            arr = getattr(p, k)
            flat = np.asarray(v, dtype=np.float64).ravel()
            for i in range(len(arr)):
                arr[i] = float(flat[i])
        elif k == "stream":
            p.stream = int(v) if v else None
        elif hasattr(p, k):
            setattr(p, k, v)
        # keys the library does not know (the oracle's neighbour_mode) are ignored
    return p


def _is_torch(x):
    return type(x).__module__.startswith("torch")


def _ptr(x):
    """(pointer, memspace, keepalive) of a numpy array or a torch tensor."""
    if _is_torch(x):
        assert x.dtype.is_floating_point and x.element_size() == 8 and x.is_contiguous()
        return x.data_ptr(), (DEVICE if x.is_cuda else HOST), x
    a = np.ascontiguousarray(x, dtype=np.float64)
    return a.ctypes.data, HOST, a


class Ccake:
    """Thin handle: every method is one ccake_* call."""

    def __init__(self, **params):
        self.params = make_params(**params)
        self._h = C.c_void_p()
        rc = lib().ccake_create(C.byref(self.params), C.byref(self._h))
        if rc != 0:
            raise CcakeError("ccake_create", rc, "(no usable CUDA device / bad parameters)")
        self.n = 0

    def _chk(self, rc, what):
        if rc != 0:
            msg = lib().ccake_last_error(self._h) if self._h else b""
            raise CcakeError(what, rc, msg.decode() if msg else "")

    def close(self):
        if self._h:
            lib().ccake_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def load_particles(self, fields: dict):
        ids = list(fields.keys())
        trip = [_ptr(fields[k]) for k in ids]
        spaces = {t[1] for t in trip}
        assert len(spaces) == 1, "all columns must live in the same memory space"
        n = int(trip[0][2].shape[0])
        assert all(int(t[2].shape[0]) == n for t in trip)
        idarr = (C.c_int32 * len(ids))(*ids)
        ptrs = (C.c_void_p * len(ids))(*[t[0] for t in trip])
        self._chk(lib().ccake_load_particles(self._h, n, len(ids), idarr, ptrs, spaces.pop()), "ccake_load_particles")
        self.n = n

    def stage_particles(self, fields: dict):
        """ccake_stage_particles: start the host -> device copies of the next particle set (pinned host columns)."""
        ids = list(fields.keys())
        trip = [_ptr(fields[k]) for k in ids]
        assert all(t[1] == HOST for t in trip)
        n = int(trip[0][2].shape[0])
        assert all(int(t[2].shape[0]) == n for t in trip)
        idarr = (C.c_int32 * len(ids))(*ids)
        ptrs = (C.c_void_p * len(ids))(*[t[0] for t in trip])
        self._chk(lib().ccake_stage_particles(self._h, n, len(ids), idarr, ptrs), "ccake_stage_particles")
        self._staged_n = n

    def load_staged(self):
        self._chk(lib().ccake_load_staged(self._h), "ccake_load_staged")
        self.n = self._staged_n

    def load_eos_table(self, axes, axis_kind, col_ids, data):
        ax = [np.ascontiguousarray(a, dtype=np.float64) for a in axes]
        dptr, space, keep = _ptr(data)
        dims = (C.c_int32 * 4)(*[len(a) for a in ax])
        kinds = (C.c_int32 * 4)(*axis_kind)
        cids = (C.c_int32 * len(col_ids))(*col_ids)
        nodes = int(np.prod([len(a) for a in ax]))
        assert int(np.prod(keep.shape)) == nodes * len(col_ids)
        if space == DEVICE:
            import torch
            axd = [torch.as_tensor(a, device=keep.device) for a in ax]
            ptrs = (C.c_void_p * 4)(*[a.data_ptr() for a in axd])
        else:
            ptrs = (C.c_void_p * 4)(*[a.ctypes.data for a in ax])
        self._chk(lib().ccake_load_eos_table(self._h, dims, kinds, ptrs, len(col_ids), cids, dptr, space),
                  "ccake_load_eos_table")

    def invert_eos_table(self, axes, axis_kind, col_ids, out=False):
        """ccake_invert_eos_table: build the conformal table on the device and install it; out=True returns it
        as a numpy array [d0, d1, d2, d3, ncols]."""
        ax = [np.ascontiguousarray(a, dtype=np.float64) for a in axes]
        dims = (C.c_int32 * 4)(*[len(a) for a in ax])
        kinds = (C.c_int32 * 4)(*axis_kind)
        cids = (C.c_int32 * len(col_ids))(*col_ids)
        ptrs = (C.c_void_p * 4)(*[a.ctypes.data for a in ax])
        res = np.empty([len(a) for a in ax] + [len(col_ids)], dtype=np.float64) if out else None
        self._chk(lib().ccake_invert_eos_table(self._h, dims, kinds, ptrs, len(col_ids), cids,
                                               res.ctypes.data if out else None, HOST), "ccake_invert_eos_table")
        return res

    def invert_forward_table(self, faxes, fdata, axes, axis_kind, col_ids, out=False):
        """ccake_invert_forward_table: invert the forward table fdata[..., 5] = (p, s, n_B, n_S, n_Q) on the (T, mu) grid
        faxes onto the (s, B, S, Q) grid axes on the device and install it.  Returns (table or None, flags, n_backup)."""
        fax = [np.ascontiguousarray(a, dtype=np.float64) for a in faxes]
        fdata = np.ascontiguousarray(fdata, dtype=np.float64)
        assert fdata.size == int(np.prod([len(a) for a in fax])) * 5
        ax = [np.ascontiguousarray(a, dtype=np.float64) for a in axes]
        fdims = (C.c_int32 * 4)(*[len(a) for a in fax])
        dims = (C.c_int32 * 4)(*[len(a) for a in ax])
        kinds = (C.c_int32 * 4)(*axis_kind)
        cids = (C.c_int32 * len(col_ids))(*col_ids)
        fptrs = (C.c_void_p * 4)(*[a.ctypes.data for a in fax])
        ptrs = (C.c_void_p * 4)(*[a.ctypes.data for a in ax])
        res = np.empty([len(a) for a in ax] + [len(col_ids)], dtype=np.float64) if out else None
        flags = np.zeros([len(a) for a in ax], dtype=np.int32)
        nb = C.c_int64(0)
        self._chk(lib().ccake_invert_forward_table(self._h, fdims, fptrs, fdata.ctypes.data, dims, kinds, ptrs, len(col_ids), cids,
                                                   res.ctypes.data if out else None, flags.ctypes.data, C.byref(nb), HOST),
                  "ccake_invert_forward_table")
        return res, flags, int(nb.value)

    def smear_sources(self, p, r, t, h_source, eta_norm=1.0):
        """ccake_smear_sources (Eq. 35): p [4, np], r [3, np], t [np] (numpy, host) -> j [4, n] numpy."""
        p = np.ascontiguousarray(p, dtype=np.float64); r = np.ascontiguousarray(r, dtype=np.float64)
        t = np.ascontiguousarray(t, dtype=np.float64)
        out = np.zeros((4, self.n), dtype=np.float64)
        pp = (C.c_void_p * 4)(*[p[m].ctypes.data for m in range(4)])
        rr = (C.c_void_p * 3)(*[r[a].ctypes.data for a in range(3)])
        oo = (C.c_void_p * 4)(*[out[m].ctypes.data for m in range(4)])
        self._chk(lib().ccake_smear_sources(self._h, t.size, pp, rr, t.ctypes.data, float(h_source), float(eta_norm),
                                            oo, HOST), "ccake_smear_sources")
        return out

    def smear_sources_noalloc(self, p, r, t, h_source, eta_norm, out):
        """ccake_smear_sources_noalloc: p (4), r (3) lists of CUDA tensors of npartons doubles, t a CUDA tensor, out a list of 4
        CUDA tensors of n doubles (overwritten).  Asynchronous: valid after synchronize().  Allocates nothing."""
        assert all(_is_torch(x) and x.is_cuda for x in list(p) + list(r) + [t] + list(out))
        pp = (C.c_void_p * 4)(*[x.data_ptr() for x in p])
        rr = (C.c_void_p * 3)(*[x.data_ptr() for x in r])
        oo = (C.c_void_p * 4)(*[x.data_ptr() for x in out])
        self._chk(lib().ccake_smear_sources_noalloc(self._h, int(t.numel()), pp, rr, t.data_ptr(), float(h_source),
                                                    float(eta_norm), oo), "ccake_smear_sources_noalloc")

    def set_sources(self, I=None, Iq=None):
        """ccake_set_sources (Eq. 38): I [4, n] contravariant I^mu, Iq [3, n] (numpy host arrays, or lists of
        CUDA tensors of n doubles); None = zero; both None switches the sources off."""
        keep = []
        space = HOST

        def ptrs(a, k):
            nonlocal space
            if a is None:
                return None
            if _is_torch(a[0]):
                space = DEVICE
                keep.extend(a)
                return (C.c_void_p * k)(*[t.data_ptr() for t in a])
            a = np.ascontiguousarray(a, dtype=np.float64).reshape(k, self.n)
            keep.append(a)
            return (C.c_void_p * k)(*[a[m].ctypes.data for m in range(k)])
        pi, pq = ptrs(I, 4), ptrs(Iq, 3)
        self._chk(lib().ccake_set_sources(self._h, pi, pq, space), "ccake_set_sources")

    def step(self, nsteps=1):
        self._chk(lib().ccake_step(self._h, nsteps), "ccake_step")

    def synchronize(self, strict=True):
        rc = lib().ccake_synchronize(self._h)
        if rc != 0 and (strict or rc != ERANGE):
            self._chk(rc, "ccake_synchronize")
        return rc

    def read_fields(self, ids, out=None):
        """Host read (numpy) by default; pass out = list of CUDA tensors for a device read."""
        ids = list(ids)
        idarr = (C.c_int32 * len(ids))(*ids)
        if out is None:
            bufs = [np.empty(self.n, dtype=np.float64) for _ in ids]
            ptrs = (C.c_void_p * len(ids))(*[b.ctypes.data for b in bufs])
            space = HOST
        else:
            bufs = list(out)
            trip = [_ptr(b) for b in bufs]
            ptrs = (C.c_void_p * len(ids))(*[t[0] for t in trip])
            space = trip[0][1]
        self._chk(lib().ccake_read_fields(self._h, len(ids), idarr, ptrs, self.n, space), "ccake_read_fields")
        return dict(zip(ids, bufs))

    def read_fields_async(self, ids, out):
        """ccake_read_fields_async into pinned host tensors / arrays `out`; valid after read_fields_wait()."""
        ids = list(ids)
        idarr = (C.c_int32 * len(ids))(*ids)
        trip = [_ptr(b) for b in out]
        assert all(t[1] == HOST for t in trip)
        ptrs = (C.c_void_p * len(ids))(*[t[0] for t in trip])
        self._chk(lib().ccake_read_fields_async(self._h, len(ids), idarr, ptrs, self.n), "ccake_read_fields_async")

    def read_fields_wait(self):
        self._chk(lib().ccake_read_fields_wait(self._h), "ccake_read_fields_wait")

    def conserved_totals(self):
        out = (C.c_double * 16)()
        self._chk(lib().ccake_conserved_totals(self._h, out), "ccake_conserved_totals")
        return np.array(out[:], dtype=np.float64)

    def read_neighbors(self):
        counts = np.empty(self.n, dtype=np.int64)
        self._chk(lib().ccake_read_neighbors(self._h, counts.ctypes.data, None, None, 0), "ccake_read_neighbors")
        offsets = np.empty(self.n + 1, dtype=np.int64)
        lst = np.empty(max(int(counts.sum()), 1), dtype=np.int32)
        self._chk(lib().ccake_read_neighbors(self._h, counts.ctypes.data, offsets.ctypes.data, lst.ctypes.data, lst.size),
                  "ccake_read_neighbors")
        return counts, offsets, lst[: int(counts.sum())]

    def neighbor_hash(self):
        out = np.empty(self.n, dtype=np.uint64)
        self._chk(lib().ccake_neighbor_hash(self._h, out.ctypes.data, self.n), "ccake_neighbor_hash")
        return out

    # ---- slab decomposition of one event (include/ccake.h, "Slab decomposition"): one call each; messages are torch
    #      device tensors of shape [29, cap] owned by the caller
    def slab_load(self, fields: dict, gids, capacity, axis, lo, hi, halo_width):
        ids = list(fields.keys())
        trip = [_ptr(fields[k]) for k in ids]
        assert {t[1] for t in trip} == {HOST}, "slab_load takes host columns"
        n = int(trip[0][2].shape[0])
        idarr = (C.c_int32 * len(ids))(*ids)
        ptrs = (C.c_void_p * len(ids))(*[t[0] for t in trip])
        g = np.ascontiguousarray(gids, dtype=np.uint32)
        assert g.size == n
        self._chk(lib().ccake_slab_load(self._h, n, int(capacity), len(ids), idarr, ptrs, g.ctypes.data, int(axis), float(lo), float(hi),
                                        float(halo_width), HOST), "ccake_slab_load")
        self.n = n

    def slab_export_halo(self, side, k, buf):
        cnt = C.c_int64(0)
        self._chk(lib().ccake_slab_export_halo(self._h, int(side), int(k), buf.data_ptr(), int(buf.shape[1]), C.byref(cnt)),
                  "ccake_slab_export_halo")
        return int(cnt.value)

    def slab_import_ghosts(self, side, k, buf, count):
        self._chk(lib().ccake_slab_import_ghosts(self._h, int(side), int(k), buf.data_ptr() if buf is not None else None,
                                                 int(buf.shape[1]) if buf is not None else 0, int(count)), "ccake_slab_import_ghosts")
        self.n = self.slab_info()[0] + self.slab_info()[1] + self.slab_info()[2]

    def slab_substep(self, k):
        self._chk(lib().ccake_slab_substep(self._h, int(k)), "ccake_slab_substep")

    def slab_substep_part(self, k, part):
        self._chk(lib().ccake_slab_substep_part(self._h, int(k), int(part)), "ccake_slab_substep_part")

    def slab_export_records(self, side, buf):
        cnt = C.c_int64(0)
        self._chk(lib().ccake_slab_export_records(self._h, int(side), buf.data_ptr(), int(buf.shape[1]), C.byref(cnt)),
                  "ccake_slab_export_records")
        return int(cnt.value)

    def slab_import_records(self, side, buf, count):
        self._chk(lib().ccake_slab_import_records(self._h, int(side), buf.data_ptr() if buf is not None else None,
                                                  int(buf.shape[1]) if buf is not None else 0, int(count)), "ccake_slab_import_records")

    def slab_export_migrants(self, side, buf):
        cnt = C.c_int64(0)
        self._chk(lib().ccake_slab_export_migrants(self._h, int(side), buf.data_ptr(), int(buf.shape[1]), C.byref(cnt)),
                  "ccake_slab_export_migrants")
        return int(cnt.value)

    def slab_import_migrants(self, side, buf, count):
        self._chk(lib().ccake_slab_import_migrants(self._h, int(side), buf.data_ptr() if buf is not None else None,
                                                   int(buf.shape[1]) if buf is not None else 0, int(count)), "ccake_slab_import_migrants")

    def slab_commit(self):
        n = C.c_int64(0)
        self._chk(lib().ccake_slab_commit(self._h, C.byref(n)), "ccake_slab_commit")
        self.n = int(n.value)
        return self.n

    def slab_info(self):
        out = (C.c_int64 * 4)()
        self._chk(lib().ccake_slab_info(self._h, out), "ccake_slab_info")
        return tuple(int(v) for v in out)

    def slab_gids(self):
        out = np.empty(self.n, dtype=np.uint32)
        self._chk(lib().ccake_slab_gids(self._h, out.ctypes.data, out.size, HOST), "ccake_slab_gids")
        return out

    def enable_timing(self, on=True):
        self._chk(lib().ccake_enable_timing(self._h, 1 if on else 0), "ccake_enable_timing")

    def launch_count(self):
        out = C.c_int64(0)
        self._chk(lib().ccake_launch_count(self._h, C.byref(out)), "ccake_launch_count")
        return int(out.value)

    def kernel_times(self):
        out = (C.c_double * 8)()
        self._chk(lib().ccake_kernel_times(self._h, out), "ccake_kernel_times")
        return np.array(out[:], dtype=np.float64)


def state_field_ids(params: dict):
    """Ids of the evolved state fields for a parameter set (what ccake_step advances)."""
    D = params["dim"]
    fl = params["flags"] if params["eom"] != 0 else 0
    ids = [R1, R2] + ([R3] if D == 3 else []) + [U1, U2] + ([U3] if D == 3 else []) + [S, NB, NS, NQ]
    if fl & 2:
        ids.append(BULK)
    if fl & 1:
        ids += [PI11, PI12, PI22, PI33] + ([PI13, PI23] if D == 3 else [])
    if fl & 4:
        ids += [JB1 + 3 * q + j for q in range(3) for j in range(D)]
    return ids


def from_workload(w, device=0, stream=None, memspace="host") -> Ccake:
    """Create a context for a paper_2511_22852_b200.workloads.Workload and load its particles and table."""
    sim = Ccake(device=device, stream=stream, **w.params)
    if w.table is not None:
        data = w.table["data"]
        if memspace == "device":
            import torch
            data = torch.as_tensor(data, device=f"cuda:{device}")
        sim.load_eos_table(w.table["axes"], w.table["axis_kind"], w.table["col_ids"], data)
    fields = w.fields
    if memspace == "device":
        import torch
        fields = {k: torch.as_tensor(np.ascontiguousarray(v), device=f"cuda:{device}") for k, v in fields.items()}
    sim.load_particles(fields)
    return sim
