"""ORACLE binding -- test infrastructure, not the product.

ctypes marshalling for ``oracle/psg_oracle.c`` (plain fp64 C, see its header).
Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline``
/ ``--impl reference`` legs may import this package.  It imports nothing from
``paper_2301_04835_b200`` and shares no code with the CUDA path.

All floating-point results are returned as float64 numpy arrays.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "psg_oracle.c")
_SO = os.path.join(_HERE, "libpsg_oracle.so")

DISTANCE, ANGLE, DIHEDRAL, COMPONENT, RGYR, DISPLACEMENT = 1, 2, 3, 4, 5, 6
PRINCIPAL_MOMENT, ASPHERICITY, ACYLINDRICITY, SHAPE_ANISOTROPY = 7, 8, 9, 10     # gyration-tensor shape CVs (R-SHAPE)
_NGROUPS = {DISTANCE: 2, ANGLE: 3, DIHEDRAL: 4, COMPONENT: 1, RGYR: 1, DISPLACEMENT: 2,
            PRINCIPAL_MOMENT: 1, ASPHERICITY: 1, ACYLINDRICITY: 1, SHAPE_ANISOTROPY: 1}


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, no contraction, no fast-math)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c99", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC",
               "-shared", _SRC, "-o", _SO + ".tmp", "-lm"]
        subprocess.check_call(cmd)
        os.replace(_SO + ".tmp", _SO)
    return _SO


class _CV(C.Structure):
    _fields_ = [("type", C.c_int), ("n_groups", C.c_int), ("is_range", C.c_int * 4),
                ("slot_begin", C.c_int * 4), ("slot_size", C.c_int * 4),
                ("range_begin", C.c_longlong * 4), ("range_size", C.c_longlong * 4),
                ("axis", C.c_int), ("period", C.c_double)]


class _Layout(C.Structure):
    _fields_ = [("n_replicas", C.c_int), ("n_atoms", C.c_longlong), ("replica_stride_atoms", C.c_longlong),
                ("pos_stride", C.c_int), ("n_cv", C.c_int), ("n_slots", C.c_int), ("per_replica_slots", C.c_int),
                ("box", C.c_double * 3)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_jac_rows.restype = C.c_longlong
        _lib.orc_deposit_hills.restype = C.c_longlong
        _lib.orc_num_threads.restype = C.c_int
    return _lib


def num_threads() -> int:
    return int(lib().orc_num_threads())


def set_threads(n: int) -> None:
    lib().orc_set_threads(C.c_int(n))


def _p(a, ty):
    return None if a is None else a.ctypes.data_as(C.POINTER(ty))


def _f32(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float32)


def _f64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def _i32(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.int32)


class System:
    """CV definitions + array layout, in the oracle's own structs.

    ``cvs``: list of dicts ``{"type": DISTANCE|..., "groups": [g, ...], "axis": int, "period": float}``
    where a group is ``("slots", begin, size)`` (a slice of the slot list) or
    ``("range", first_atom, n_atoms)``.
    ``slot_atom``: int32 ``[n_slots]`` (shared) or ``[R][n_slots]`` (per replica), 0-based.
    """

    def __init__(self, n_replicas, n_atoms, replica_stride_atoms, pos_stride, cvs, slot_atom,
                 slot_weight=None, atom_weight=None, box=None):
        self.cvs_py = cvs
        self.n_cv = len(cvs)
        arr = (_CV * self.n_cv)()
        for k, cv in enumerate(cvs):
            arr[k].type = cv["type"]
            arr[k].n_groups = len(cv["groups"])
            assert arr[k].n_groups == _NGROUPS[cv["type"]]
            for g, grp in enumerate(cv["groups"]):
                if grp[0] == "range":
                    arr[k].is_range[g] = 1
                    arr[k].range_begin[g] = int(grp[1])
                    arr[k].range_size[g] = int(grp[2])
                else:
                    arr[k].is_range[g] = 0
                    arr[k].slot_begin[g] = int(grp[1])
                    arr[k].slot_size[g] = int(grp[2])
            arr[k].axis = int(cv.get("axis", 0))
            arr[k].period = float(cv.get("period", 0.0))
        self.cvs = arr
        self.slot_atom = _i32(slot_atom if slot_atom is not None else np.zeros(0, np.int32))
        per_rep = 1 if self.slot_atom.ndim == 2 else 0
        n_slots = self.slot_atom.shape[-1] if self.slot_atom.size else 0
        self.layout = _Layout(int(n_replicas), int(n_atoms), int(replica_stride_atoms), int(pos_stride),
                              self.n_cv, int(n_slots), per_rep)
        for x in range(3):      # orthorhombic box lengths for the minimum-image convention; 0 = open (reading R-MI)
            self.layout.box[x] = float(box[x]) if box is not None else 0.0
        self.slot_weight = _f32(slot_weight)
        self.atom_weight = _f32(atom_weight)
        self.R = int(n_replicas)
        self.N = int(n_atoms)
        self.shared = replica_stride_atoms == 0
        self.period = np.array([float(cv.get("period", 0.0)) for cv in cvs], dtype=np.float64)
        self.jac_rows = int(lib().orc_jac_rows(C.byref(self.layout), self.cvs))

    def cv_eval(self, pos, want_jac=True):
        """xi [R][n_cv]; jac [R][jac_rows][3] (rows: CV by CV, group by group, atom by atom)."""
        pos = _f32(pos)
        xi = np.empty((self.R, self.n_cv), np.float64)
        jac = np.zeros((self.R, self.jac_rows, 3), np.float64) if want_jac else None
        lib().orc_cv_eval(C.byref(self.layout), self.cvs, _p(self.slot_atom, C.c_int),
                          _p(self.slot_weight, C.c_float), _p(self.atom_weight, C.c_float),
                          _p(pos, C.c_float), _p(xi, C.c_double), _p(jac, C.c_double))
        return (xi, jac) if want_jac else xi

    def abf_estimate(self, pos, vel, mass, dt, fbias_prev, whist, first):
        """ABF instantaneous-force estimator (reading R-ABF-EST): returns (fsample [R][n_cv], W [R][n_cv]); ``whist``
        [R][2][n_cv] float64 is advanced in place; ``fbias_prev`` [R][n_cv] or None."""
        pos, vel, mass = _f32(pos), _f32(vel), _f32(mass)
        assert whist.dtype == np.float64 and whist.flags.c_contiguous and whist.shape == (self.R, 2, self.n_cv)
        fb = None if fbias_prev is None else _f64(fbias_prev)
        fs = np.empty((self.R, self.n_cv), np.float64)
        w = np.empty((self.R, self.n_cv), np.float64)
        lib().orc_abf_estimate(C.byref(self.layout), self.cvs, _p(self.slot_atom, C.c_int), _p(self.slot_weight, C.c_float),
                               _p(self.atom_weight, C.c_float), _p(pos, C.c_float), _p(vel, C.c_float), _p(mass, C.c_float),
                               C.c_double(float(dt)), _p(fb, C.c_double), _p(whist, C.c_double), C.c_int(1 if first else 0),
                               _p(fs, C.c_double), _p(w, C.c_double))
        return fs, w

    def apply_forces(self, pos, dVdxi, force):
        """force: fp64 [n_arrays][N][3] (n_arrays = 1 if shared else R); returns the updated copy."""
        pos = _f32(pos)
        dv = _f64(dVdxi)
        f = np.array(force, dtype=np.float64, order="C", copy=True)
        lib().orc_apply_forces(C.byref(self.layout), self.cvs, _p(self.slot_atom, C.c_int),
                               _p(self.slot_weight, C.c_float), _p(self.atom_weight, C.c_float),
                               _p(pos, C.c_float), _p(dv, C.c_double), _p(f, C.c_double))
        return f


def harmonic(xi, kspring, center, period):
    xi = _f64(xi)
    R, n_cv = xi.shape
    V = np.empty(R, np.float64)
    dV = np.empty((R, n_cv), np.float64)
    lib().orc_harmonic(C.c_int(R), C.c_int(n_cv), _p(xi, C.c_double), _p(_f64(kspring), C.c_double),
                       _p(_f64(center), C.c_double), _p(_f64(period), C.c_double),
                       _p(V, C.c_double), _p(dV, C.c_double))
    return V, dV


def metad(xi, centers, heights, sigma, period):
    """V [R], dVdxi [R][n_cv], Tabs [R][n_cv] (sum of |gradient terms|)."""
    xi = _f64(xi)
    R, n_cv = xi.shape
    centers = _f32(centers).reshape(-1, n_cv)
    heights = _f32(heights)
    n_h = heights.shape[0]
    V = np.empty(R, np.float64)
    dV = np.empty((R, n_cv), np.float64)
    T = np.empty((R, n_cv), np.float64)
    lib().orc_metad(C.c_int(R), C.c_int(n_cv), _p(xi, C.c_double), C.c_longlong(n_h),
                    _p(centers, C.c_float), _p(heights, C.c_float), _p(_f64(sigma), C.c_double),
                    _p(_f64(period), C.c_double), _p(V, C.c_double), _p(dV, C.c_double), _p(T, C.c_double))
    return V, dV, T


def deposit_hills(xi_f32, mask, w0, kB_deltaT, sigma, period, n_hills, centers, heights):
    """Append in place to ``centers`` [cap][n_cv] / ``heights`` [cap] (float32); returns new count."""
    xi = _f32(xi_f32)
    R, n_cv = xi.shape
    assert centers.dtype == np.float32 and heights.dtype == np.float32
    assert centers.flags.c_contiguous and heights.flags.c_contiguous
    m = None if mask is None else np.ascontiguousarray(mask, dtype=np.uint8)
    n_dep = R if m is None else int(m.astype(bool).sum())
    assert n_hills + n_dep <= heights.shape[0], "hill store capacity"
    return int(lib().orc_deposit_hills(C.c_int(R), C.c_int(n_cv), _p(xi, C.c_float), _p(m, C.c_ubyte),
                                       C.c_double(w0), C.c_double(kB_deltaT), _p(_f64(sigma), C.c_double),
                                       _p(_f64(period), C.c_double), C.c_longlong(n_hills),
                                       _p(centers, C.c_float), _p(heights, C.c_float)))


def abf_update(xi_f32, fsample_f32, lower, upper, shape, periodic, n_threshold, hist, fsum):
    """Updates ``hist`` (int32 [nbins]) and ``fsum`` (float64 [nbins][n_cv]) in place.
    Returns bin [R] int32 and dVdxi [R][n_cv] float64."""
    xi = _f32(xi_f32)
    R, n_cv = xi.shape
    assert hist.dtype == np.int32 and fsum.dtype == np.float64
    b = np.empty(R, np.int32)
    dV = np.empty((R, n_cv), np.float64)
    lib().orc_abf_update(C.c_int(R), C.c_int(n_cv), _p(xi, C.c_float), _p(_f32(fsample_f32), C.c_float),
                         _p(_f32(lower), C.c_float), _p(_f32(upper), C.c_float), _p(_i32(shape), C.c_int),
                         _p(_i32(periodic), C.c_int), C.c_int(n_threshold), _p(hist, C.c_int),
                         _p(fsum, C.c_double), _p(b, C.c_int), _p(dV, C.c_double))
    return b, dV


def dist_to_interface(pos, mobile_idx, mobile_w, ibegin, n_i, axis, sigma, scope, bins, coeff):
    """DistanceToInterface of ONE replica (Sec. 2.2.1 / App. A): pos float32 [N][stride].
    Returns (xi, jac_mobile [n_m][3], dxi_dx [n_i], mass [bins])."""
    pos = _f32(pos)
    idx = _i32(np.asarray(mobile_idx))
    wm = _f32(mobile_w)
    xi = C.c_double(0.0)
    jm = np.zeros((len(idx), 3), np.float64)
    dx = np.zeros(int(n_i), np.float64)
    mass = np.zeros(int(bins), np.float64)
    lib().orc_dist_to_interface(_p(pos, C.c_float), C.c_int(pos.shape[-1]), C.c_int(len(idx)), _p(idx, C.c_int), _p(wm, C.c_float),
                                C.c_longlong(int(ibegin)), C.c_longlong(int(n_i)), C.c_int(int(axis)), C.c_double(float(sigma)),
                                C.c_double(float(scope[0])), C.c_double(float(scope[1])), C.c_int(int(bins)), C.c_double(float(coeff)),
                                C.byref(xi), _p(jm, C.c_double), _p(dx, C.c_double), _p(mass, C.c_double))
    return xi.value, jm, dx, mass


class _Grid(C.Structure):
    _fields_ = [("n_cv", C.c_int), ("lower", C.c_double * 4), ("upper", C.c_double * 4), ("shape", C.c_int * 4),
                ("periodic", C.c_int * 4)]


class MetadGrid:
    """Grid-stored metadynamics (reading R-GRID).  ``values`` is the node array
    [nodes][1 + n_cv] (V, dV/dxi_1, ...), float64, row-major with the last CV fastest; tests may write it directly."""

    def __init__(self, lower, upper, shape, periodic):
        self.g = _Grid()
        self.n_cv = self.g.n_cv = len(shape)
        for k in range(self.n_cv):
            self.g.lower[k], self.g.upper[k] = float(lower[k]), float(upper[k])
            self.g.shape[k], self.g.periodic[k] = int(shape[k]), int(bool(periodic[k]))
        lib().orc_grid_nodes.restype = C.c_longlong
        self.nodes = int(lib().orc_grid_nodes(C.byref(self.g)))
        self.values = np.zeros((self.nodes, 1 + self.n_cv), np.float64)

    def eval(self, xi):
        xi = _f64(xi).reshape(-1, self.n_cv)
        V = np.empty(xi.shape[0], np.float64)
        dV = np.empty((xi.shape[0], self.n_cv), np.float64)
        lib().orc_grid_eval(C.byref(self.g), _p(self.values, C.c_double), C.c_int(xi.shape[0]), _p(xi, C.c_double),
                            _p(V, C.c_double), _p(dV, C.c_double))
        return V, dV

    def deposit(self, xi_f32, sigma, w0, kB_deltaT=0.0, mask=None):
        """one synchronous deposit event; returns the heights [R] (0 where masked out)"""
        xi = _f32(xi_f32).reshape(-1, self.n_cv)
        m = None if mask is None else np.ascontiguousarray(mask, dtype=np.uint8)
        h = np.empty(xi.shape[0], np.float64)
        lib().orc_grid_deposit(C.byref(self.g), _p(self.values, C.c_double), C.c_int(xi.shape[0]), _p(xi, C.c_float),
                               _p(m, C.c_ubyte), C.c_double(w0), C.c_double(kB_deltaT), _p(_f64(sigma), C.c_double),
                               _p(h, C.c_double))
        return h
