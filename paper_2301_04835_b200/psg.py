"""ctypes marshalling for libpsg.so.  Method names are the C names without the ``psg_`` prefix
(include/psg.h documents every call).  Tensors are torch CUDA tensors (float32 / int32 /
uint8, contiguous); only their ``data_ptr()`` crosses the boundary.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libpsg.so")

CV_DISTANCE, CV_ANGLE, CV_DIHEDRAL, CV_COM_COMPONENT, CV_RGYR, CV_DISPLACEMENT = 1, 2, 3, 4, 5, 6
CV_PRINCIPAL_MOMENT, CV_ASPHERICITY, CV_ACYLINDRICITY, CV_SHAPE_ANISOTROPY, CV_DIST_TO_INTERFACE = 7, 8, 9, 10, 11
METHOD_NONE, METHOD_HARMONIC, METHOD_METAD, METHOD_ABF, METHOD_METAD_GRID = 0, 1, 2, 3, 4
HILLS_F32, HILLS_F64 = 0, 1
_KIND = {"distance": CV_DISTANCE, "angle": CV_ANGLE, "dihedral": CV_DIHEDRAL, "component": CV_COM_COMPONENT,
         "rgyr": CV_RGYR, "displacement": CV_DISPLACEMENT, "principal_moment": CV_PRINCIPAL_MOMENT,
         "asphericity": CV_ASPHERICITY, "acylindricity": CV_ACYLINDRICITY, "shape_anisotropy": CV_SHAPE_ANISOTROPY,
         "dist_to_interface": CV_DIST_TO_INTERFACE}

# every symbol include/psg.h declares
EXPORTS = ["psg_create", "psg_destroy", "psg_set_stream", "psg_last_error", "psg_set_layout", "psg_set_cvs",
           "psg_set_box", "psg_set_harmonic", "psg_set_metad", "psg_set_hill_precision", "psg_load_hills", "psg_get_hills",
           "psg_set_abf", "psg_abf_state", "psg_cv_eval", "psg_bias_eval", "psg_deposit_hill", "psg_abf_update",
           "psg_abf_accumulate_delta", "psg_abf_apply_grid_delta", "psg_abf_estimate", "psg_abf_estimate_reset", "psg_apply_bias_forces", "psg_step", "psg_step_outputs", "psg_step_host", "psg_sync_check",
           "psg_interface_cv_set", "psg_interface_cv_eval", "psg_interface_cv_apply", "psg_hill_heights", "psg_append_hills", "psg_set_metad_grid", "psg_metad_grid_set",
           "psg_metad_grid_deposit", "psg_metad_grid_eval", "psg_metad_grid_step", "psg_metad_grid_state", "psg_measure_alu_peak", "psg_launch_count", "psg_set_tuning",
           "psg_range_rgyr_static", "psg_static_last_error"]


class PsgError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libpsg error {code}: {msg}")
        self.code = code


class _CvDesc(C.Structure):
    _fields_ = [("type", C.c_int), ("n_groups", C.c_int), ("group_is_range", C.c_int * 4),
                ("group_begin", C.c_int * 4), ("group_size", C.c_int * 4),
                ("range_begin", C.c_longlong * 4), ("range_size", C.c_longlong * 4),
                ("axis", C.c_int), ("period", C.c_double), ("dti_sigma", C.c_double), ("dti_scope", C.c_double * 2),
                ("dti_coeff", C.c_double), ("dti_bins", C.c_int)]


_lib = None


def lib_path() -> str:
    return _LIB_PATH


def load_library():
    """dlopen libpsg.so (built in-tree by ``python -m paper_2301_04835_b200.build``). Fails loudly if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise PsgError(-3, f"{_LIB_PATH} is missing: run `python -m paper_2301_04835_b200.build` "
                               "(there is no CPU fallback)")
        L = C.CDLL(_LIB_PATH)
        L.psg_last_error.restype = C.c_char_p
        L.psg_last_error.argtypes = [C.c_void_p]
        L.psg_launch_count.restype = C.c_longlong
        L.psg_launch_count.argtypes = [C.c_void_p]
        vp, i, ll, f = C.c_void_p, C.c_int, C.c_longlong, C.c_float
        L.psg_create.argtypes = [C.POINTER(vp), i, vp]
        L.psg_destroy.argtypes = [vp]
        L.psg_set_stream.argtypes = [vp, vp]
        L.psg_set_layout.argtypes = [vp, i, ll, ll, i, i]
        L.psg_set_cvs.argtypes = [vp, i, C.POINTER(_CvDesc), i, vp, i, vp, vp]
        L.psg_set_box.argtypes = [vp, vp]
        L.psg_set_harmonic.argtypes = [vp, vp, vp]
        L.psg_set_metad.argtypes = [vp, vp, f, f, i, i]
        L.psg_set_hill_precision.argtypes = [vp, i]
        L.psg_load_hills.argtypes = [vp, i, vp, vp]
        L.psg_get_hills.argtypes = [vp, C.POINTER(i), vp, vp, i]
        L.psg_set_abf.argtypes = [vp, vp, vp, vp, vp, i, vp, vp]
        L.psg_abf_state.argtypes = [vp, C.POINTER(vp), C.POINTER(vp), C.POINTER(ll)]
        L.psg_cv_eval.argtypes = [vp, vp, vp, vp]
        L.psg_bias_eval.argtypes = [vp, vp, vp, vp]
        L.psg_deposit_hill.argtypes = [vp, vp, vp]
        L.psg_abf_update.argtypes = [vp, vp, vp, vp, vp]
        L.psg_abf_accumulate_delta.argtypes = [vp, vp, vp, vp, vp]
        L.psg_abf_apply_grid_delta.argtypes = [vp, vp, vp, vp, vp]
        L.psg_abf_estimate.argtypes = [vp, vp, vp, vp, C.c_double, vp, vp]
        L.psg_abf_estimate_reset.argtypes = [vp]
        L.psg_apply_bias_forces.argtypes = [vp, vp, vp, vp]
        L.psg_step.argtypes = [vp, vp, vp, vp, ll]
        L.psg_step_outputs.argtypes = [vp, C.POINTER(vp), C.POINTER(vp), C.POINTER(vp), C.POINTER(vp)]
        L.psg_step_host.argtypes = [vp, vp, vp, vp, ll]
        L.psg_sync_check.argtypes = [vp]
        d = C.c_double
        L.psg_interface_cv_set.argtypes = [vp, i, vp, vp, ll, ll, i, d, d, d, i, d]
        L.psg_interface_cv_eval.argtypes = [vp, vp, vp]
        L.psg_interface_cv_apply.argtypes = [vp, vp, vp, vp]
        L.psg_hill_heights.argtypes = [vp, vp, vp, vp]
        L.psg_append_hills.argtypes = [vp, i, vp, vp]
        L.psg_metad_grid_set.argtypes = [vp, i, vp, vp, vp, vp, vp, d, d]
        L.psg_set_metad_grid.argtypes = [vp, vp, vp, vp, vp, vp, d, d, i]
        L.psg_metad_grid_deposit.argtypes = [vp, vp, vp]
        L.psg_metad_grid_eval.argtypes = [vp, vp, vp, vp]
        L.psg_metad_grid_state.argtypes = [vp, vp, vp, vp]
        L.psg_metad_grid_step.argtypes = [vp, vp, vp]
        L.psg_measure_alu_peak.argtypes = [i, i, C.POINTER(C.c_double)]
        L.psg_set_tuning.argtypes = [vp, i, i]
        L.psg_range_rgyr_static.argtypes = [i, vp, vp, i, i, ll, ll, ll, vp, vp, vp]
        L.psg_static_last_error.restype = C.c_char_p
        L.psg_static_last_error.argtypes = []
        _lib = L
    return _lib


def _dp(t, dtype=None):
    """device pointer of a torch CUDA tensor (None -> NULL)"""
    if t is None:
        return None
    if not t.is_cuda or not t.is_contiguous():
        raise ValueError("expected a contiguous CUDA tensor")
    if dtype is not None and t.dtype != dtype:
        raise ValueError(f"expected dtype {dtype}, got {t.dtype}")
    return C.c_void_p(t.data_ptr())


def _hp(a, dtype):
    """host pointer of a numpy array (None -> NULL); returns (keepalive, pointer)"""
    if a is None:
        return None, None
    a = np.ascontiguousarray(a, dtype=dtype)
    return a, C.c_void_p(a.ctypes.data)


def measure_alu_peak(which: int, device: int = 0) -> float:
    out = C.c_double(0.0)
    rc = load_library().psg_measure_alu_peak(device, which, C.byref(out))
    if rc != 0:
        raise PsgError(rc, "psg_measure_alu_peak failed")
    return out.value


def range_rgyr_static(pos, first_atom, n_group_atoms, weight=None, xi=None, center=None, device=0, stream=None):
    """psg_range_rgyr_static (include/psg_static.h): radius of gyration of one contiguous atom range per replica, with no
    allocation inside the library (static device scratch; limit PSG_STATIC_MAX_BLOCKS).  pos: CUDA float32 [R][stride][3|4];
    weight: CUDA float32 [>= first + n] or None; xi: CUDA float32 [R] out; center: CUDA float64 [R][4] out or None.
    stream: raw cudaStream_t, torch.cuda.Stream or None = torch's current stream.  Argument marshalling only."""
    import torch
    if stream is None:
        stream = torch.cuda.current_stream(device).cuda_stream
    elif hasattr(stream, "cuda_stream"):
        stream = stream.cuda_stream
    if pos.dim() != 3 or xi is None:
        raise ValueError("pos must be [R][stride][3|4] and xi [R] must be given (this call allocates nothing)")
    L = load_library()
    rc = L.psg_range_rgyr_static(device, C.c_void_p(stream), _dp(pos, torch.float32), pos.shape[2], pos.shape[0], pos.shape[1],
                                 int(first_atom), int(n_group_atoms), _dp(weight, torch.float32), _dp(xi, torch.float32),
                                 _dp(center, torch.float64))
    if rc != 0:
        raise PsgError(rc, L.psg_static_last_error().decode())
    return xi


class Context:
    """One psg_ctx.  ``stream``: a raw cudaStream_t (int), a torch.cuda.Stream, or None = torch's current stream."""

    def __init__(self, device: int = 0, stream=None):
        import torch
        self._torch = torch
        self._L = load_library()
        self._h = C.c_void_p()
        self.device = device
        if stream is None:
            stream = torch.cuda.current_stream(device).cuda_stream
        elif hasattr(stream, "cuda_stream"):
            stream = stream.cuda_stream
        rc = self._L.psg_create(C.byref(self._h), device, C.c_void_p(stream))
        if rc != 0:
            raise PsgError(rc, self._L.psg_last_error(None).decode())
        self.stream_handle = int(stream or 0)      # the cudaStream_t the ctx enqueues on (multiwalker orders collectives against it)
        self.R = self.n_cv = self.n_slots = 0

    def _ck(self, rc):
        if rc != 0:
            raise PsgError(rc, self._L.psg_last_error(self._h).decode())

    def close(self):
        if self._h:
            self._L.psg_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ------------------------------------------------------------------ setup
    def set_stream(self, stream):
        if hasattr(stream, "cuda_stream"):
            stream = stream.cuda_stream
        self._ck(self._L.psg_set_stream(self._h, C.c_void_p(stream)))
        self.stream_handle = int(stream or 0)

    def set_layout(self, n_replicas, n_atoms, replica_stride_atoms, pos_stride_floats=4, frc_stride_floats=4):
        self._ck(self._L.psg_set_layout(self._h, n_replicas, n_atoms, replica_stride_atoms, pos_stride_floats,
                                        frc_stride_floats))
        self.R = n_replicas

    def set_cvs(self, cvs, slot_atom_idx=None, slot_weight=None, atom_weight=None):
        """cvs: list of dicts {"type": CV_*, "groups": [("slots", begin, size) | ("range", first, n)], "axis", "period"[, "dti"]}"""
        arr = (_CvDesc * len(cvs))()
        for k, cv in enumerate(cvs):
            arr[k].type = cv["type"]
            arr[k].n_groups = len(cv["groups"])
            for g, grp in enumerate(cv["groups"]):
                if grp[0] == "range":
                    arr[k].group_is_range[g] = 1
                    arr[k].range_begin[g], arr[k].range_size[g] = int(grp[1]), int(grp[2])
                else:
                    arr[k].group_begin[g], arr[k].group_size[g] = int(grp[1]), int(grp[2])
            arr[k].axis = int(cv.get("axis", 0))
            arr[k].period = float(cv.get("period", 0.0))
            if "dti" in cv:     # {"sigma", "scope": (lo, hi), "bins", "coeff"} of PSG_CV_DIST_TO_INTERFACE
                d = cv["dti"]
                arr[k].dti_sigma, arr[k].dti_coeff, arr[k].dti_bins = float(d["sigma"]), float(d["coeff"]), int(d["bins"])
                arr[k].dti_scope[0], arr[k].dti_scope[1] = float(d["scope"][0]), float(d["scope"][1])
        if slot_atom_idx is None:
            sa, n_slots, per_rep = None, 0, 0
        else:
            sa = np.ascontiguousarray(slot_atom_idx, dtype=np.int32)
            n_slots, per_rep = sa.shape[-1], int(sa.ndim == 2)
        k1, p_sa = _hp(sa, np.int32)
        k2, p_sw = _hp(slot_weight, np.float32)
        k3, p_aw = _hp(atom_weight, np.float32)
        self._ck(self._L.psg_set_cvs(self._h, len(cvs), arr, n_slots, p_sa, per_rep, p_sw, p_aw))
        self.n_cv, self.n_slots = len(cvs), n_slots

    def set_box(self, box):
        """orthorhombic box lengths [3] for the minimum-image convention (0 = open); None switches it off"""
        k1, p1 = _hp(None if box is None else np.asarray(box, np.float64), np.float64)
        self._ck(self._L.psg_set_box(self._h, p1))

    def set_harmonic(self, kspring, centers):
        k1, p1 = _hp(kspring, np.float32)
        k2, p2 = _hp(centers, np.float32)
        self._ck(self._L.psg_set_harmonic(self._h, p1, p2))

    def set_metad(self, sigma, w0, kB_deltaT, capacity, stride=0):
        k1, p1 = _hp(sigma, np.float32)
        self._ck(self._L.psg_set_metad(self._h, p1, float(w0), float(kB_deltaT), int(capacity), int(stride)))

    def set_hill_precision(self, mode):
        self._ck(self._L.psg_set_hill_precision(self._h, mode))

    def hill_heights(self, d_xi, d_mask, d_heights):
        t = self._torch
        self._ck(self._L.psg_hill_heights(self._h, _dp(d_xi, t.float32), _dp(d_mask, t.uint8), _dp(d_heights, t.float32)))

    def append_hills(self, d_centers, d_heights):
        t = self._torch
        n = int(d_heights.shape[0])
        self._ck(self._L.psg_append_hills(self._h, n, _dp(d_centers, t.float32), _dp(d_heights, t.float32)))

    def load_hills(self, d_centers, d_heights):
        n = int(d_heights.shape[0]) if d_heights is not None else 0
        t = self._torch
        self._ck(self._L.psg_load_hills(self._h, n, _dp(d_centers, t.float32), _dp(d_heights, t.float32)))

    def get_hills(self):
        """(centers [n][n_cv], heights [n]) as new CUDA tensors; synchronises."""
        t = self._torch
        n = C.c_int(0)
        self._ck(self._L.psg_get_hills(self._h, C.byref(n), None, None, 0))
        c = t.empty((n.value, self.n_cv), dtype=t.float32, device=f"cuda:{self.device}")
        h = t.empty((n.value,), dtype=t.float32, device=f"cuda:{self.device}")
        self._ck(self._L.psg_get_hills(self._h, C.byref(n), _dp(c), _dp(h), n.value))
        return c, h

    def n_hills(self):
        n = C.c_int(0)
        self._ck(self._L.psg_get_hills(self._h, C.byref(n), None, None, 0))
        return n.value

    def set_abf(self, lower, upper, shape, periodic, n_threshold, d_hist=None, d_fsum=None):
        t = self._torch
        k1, p1 = _hp(lower, np.float32)
        k2, p2 = _hp(upper, np.float32)
        k3, p3 = _hp(shape, np.int32)
        k4, p4 = _hp(periodic, np.int32)
        self._abf_keep = (d_hist, d_fsum)
        self._ck(self._L.psg_set_abf(self._h, p1, p2, p3, p4, int(n_threshold), _dp(d_hist, t.int32),
                                     _dp(d_fsum, t.float32)))

    def abf_state(self):
        """(hist_ptr, fsum_ptr, n_bins) raw device pointers of the grid in use"""
        h, f, n = C.c_void_p(), C.c_void_p(), C.c_longlong()
        self._ck(self._L.psg_abf_state(self._h, C.byref(h), C.byref(f), C.byref(n)))
        return h.value, f.value, n.value

    # --------------------------------------------------------------- hot path
    def cv_eval(self, d_pos, d_xi, d_jac=None):
        t = self._torch
        self._ck(self._L.psg_cv_eval(self._h, _dp(d_pos, t.float32), _dp(d_xi, t.float32), _dp(d_jac, t.float32)))

    def bias_eval(self, d_xi, d_V, d_dVdxi):
        t = self._torch
        self._ck(self._L.psg_bias_eval(self._h, _dp(d_xi, t.float32), _dp(d_V, t.float32), _dp(d_dVdxi, t.float32)))

    def deposit_hill(self, d_xi, d_mask=None):
        t = self._torch
        self._ck(self._L.psg_deposit_hill(self._h, _dp(d_xi, t.float32), _dp(d_mask, t.uint8)))

    def abf_update(self, d_xi, d_fsample, d_bin, d_dVdxi):
        t = self._torch
        self._ck(self._L.psg_abf_update(self._h, _dp(d_xi, t.float32), _dp(d_fsample, t.float32), _dp(d_bin, t.int32),
                                        _dp(d_dVdxi, t.float32)))

    def abf_accumulate_delta(self, d_pos, d_fsample, d_hist_delta, d_fsum_delta):
        t = self._torch
        self._ck(self._L.psg_abf_accumulate_delta(self._h, _dp(d_pos, t.float32), _dp(d_fsample, t.float32),
                                                  _dp(d_hist_delta, t.int32), _dp(d_fsum_delta, t.float32)))

    def abf_apply_grid_delta(self, d_hist_delta, d_fsum_delta, d_pos, d_force):
        t = self._torch
        self._ck(self._L.psg_abf_apply_grid_delta(self._h, _dp(d_hist_delta, t.int32), _dp(d_fsum_delta, t.float32),
                                                  _dp(d_pos, t.float32), _dp(d_force, t.float32)))

    def abf_n_bins(self):
        return int(self.abf_state()[2])

    def abf_estimate(self, d_pos, d_vel, d_mass, dt, d_fbias_prev, d_fsample):
        t = self._torch
        self._ck(self._L.psg_abf_estimate(self._h, _dp(d_pos, t.float32), _dp(d_vel, t.float32), _dp(d_mass, t.float32),
                                          float(dt), _dp(d_fbias_prev, t.float32), _dp(d_fsample, t.float32)))

    def abf_estimate_reset(self):
        self._ck(self._L.psg_abf_estimate_reset(self._h))

    def apply_bias_forces(self, d_pos, d_dVdxi, d_force):
        t = self._torch
        self._ck(self._L.psg_apply_bias_forces(self._h, _dp(d_pos, t.float32), _dp(d_dVdxi, t.float32),
                                               _dp(d_force, t.float32)))

    def step(self, d_pos, d_force, d_fsample=None, step=0):
        t = self._torch
        self._ck(self._L.psg_step(self._h, _dp(d_pos, t.float32), _dp(d_force, t.float32), _dp(d_fsample, t.float32),
                                  int(step)))

    def step_outputs(self):
        """raw device pointers (xi, V, dVdxi, bin) of the last step's per-replica results"""
        a, b, c, d = C.c_void_p(), C.c_void_p(), C.c_void_p(), C.c_void_p()
        self._ck(self._L.psg_step_outputs(self._h, C.byref(a), C.byref(b), C.byref(c), C.byref(d)))
        return a.value, b.value, c.value, d.value

    def step_host(self, h_pos, h_force, h_fsample=None, step=0):
        """h_pos / h_force / h_fsample: CPU tensors (pinned recommended) or numpy float32 arrays"""
        def hp(x):
            if x is None:
                return None
            if isinstance(x, np.ndarray):
                assert x.dtype == np.float32 and x.flags.c_contiguous
                return C.c_void_p(x.ctypes.data)
            assert (not x.is_cuda) and x.is_contiguous() and x.dtype == self._torch.float32
            return C.c_void_p(x.data_ptr())
        self._ck(self._L.psg_step_host(self._h, hp(h_pos), hp(h_force), hp(h_fsample), int(step)))

    # ---- DistanceToInterface (Sec. 2.2.1, App. A)
    def interface_cv_set(self, mobile_idx, mobile_w, iface_begin, iface_size, axis, sigma, scope, bins, coeff):
        k1, p1 = _hp(np.asarray(mobile_idx), np.int32)
        k2, p2 = _hp(None if mobile_w is None else np.asarray(mobile_w), np.float32)
        self._ck(self._L.psg_interface_cv_set(self._h, len(k1), p1, p2, int(iface_begin), int(iface_size), int(axis), float(sigma),
                                              float(scope[0]), float(scope[1]), int(bins), float(coeff)))

    def interface_cv_eval(self, d_pos, d_xi):
        t = self._torch
        self._ck(self._L.psg_interface_cv_eval(self._h, _dp(d_pos, t.float32), _dp(d_xi, t.float32)))

    def interface_cv_apply(self, d_pos, d_dVdxi, d_force):
        t = self._torch
        self._ck(self._L.psg_interface_cv_apply(self._h, _dp(d_pos, t.float32), _dp(d_dVdxi, t.float32), _dp(d_force, t.float32)))

    # ---- grid-stored metadynamics
    def metad_grid_set(self, lower, upper, shape, periodic, sigma, w0, kB_deltaT=0.0):
        k1, p1 = _hp(np.asarray(lower), np.float64)
        k2, p2 = _hp(np.asarray(upper), np.float64)
        k3, p3 = _hp(np.asarray(shape), np.int32)
        k4, p4 = _hp(np.asarray(periodic), np.int32)
        k5, p5 = _hp(np.asarray(sigma), np.float64)
        self._ck(self._L.psg_metad_grid_set(self._h, len(k3), p1, p2, p3, p4, p5, float(w0), float(kB_deltaT)))

    def set_metad_grid(self, lower, upper, shape, periodic, sigma, w0, kB_deltaT=0.0, stride=0):
        """the grid-stored bias as the ctx's method: psg_step then deposits every `stride` steps and interpolates"""
        k1, p1 = _hp(np.asarray(lower), np.float64)
        k2, p2 = _hp(np.asarray(upper), np.float64)
        k3, p3 = _hp(np.asarray(shape), np.int32)
        k4, p4 = _hp(np.asarray(periodic), np.int32)
        k5, p5 = _hp(np.asarray(sigma), np.float64)
        self._ck(self._L.psg_set_metad_grid(self._h, p1, p2, p3, p4, p5, float(w0), float(kB_deltaT), int(stride)))

    def metad_grid_deposit(self, d_xi, d_mask=None):
        t = self._torch
        self._ck(self._L.psg_metad_grid_deposit(self._h, _dp(d_xi, t.float32), _dp(d_mask, t.uint8)))

    def metad_grid_eval(self, d_xi, d_V, d_dVdxi):
        t = self._torch
        self._ck(self._L.psg_metad_grid_eval(self._h, _dp(d_xi, t.float32), _dp(d_V, t.float32), _dp(d_dVdxi, t.float32)))

    def metad_grid_step(self, d_pos, d_force):
        t = self._torch
        self._ck(self._L.psg_metad_grid_step(self._h, _dp(d_pos, t.float32), _dp(d_force, t.float32)))

    def metad_grid_state(self):
        """(grid_ptr, n_nodes, heights_ptr) raw device pointers (binary64)"""
        g, n, h = C.c_void_p(), C.c_longlong(), C.c_void_p()
        self._ck(self._L.psg_metad_grid_state(self._h, C.byref(g), C.byref(n), C.byref(h)))
        return g.value, n.value, h.value

    def set_tuning(self, range_step_lag=0, disable_range_step=False):
        self._ck(self._L.psg_set_tuning(self._h, int(range_step_lag), int(bool(disable_range_step))))

    def sync_check(self):
        self._ck(self._L.psg_sync_check(self._h))

    def launch_count(self) -> int:
        return int(self._L.psg_launch_count(self._h))

    # ---- convenience: read step outputs into fresh tensors (copies; not on the hot path)
    def read_step_outputs(self):
        t = self._torch
        xi_p, V_p, dV_p, bin_p = self.step_outputs()
        out = {}
        for name, ptr, shape, dt in (("xi", xi_p, (self.R, self.n_cv), t.float32), ("V", V_p, (self.R,), t.float32),
                                     ("dVdxi", dV_p, (self.R, self.n_cv), t.float32), ("bin", bin_p, (self.R,), t.int32)):
            if not ptr:
                continue
            out[name] = _view(ptr, shape, dt, self.device).clone()
        return out


class _DevView:
    """zero-copy view of ctx-owned device memory through __cuda_array_interface__"""

    def __init__(self, ptr, shape, typestr):
        self.__cuda_array_interface__ = {"shape": tuple(shape), "typestr": typestr, "data": (int(ptr), False),
                                         "version": 2, "strides": None}


def _view(ptr, shape, dtype, device):
    import torch
    typestr = {torch.float32: "<f4", torch.int32: "<i4", torch.float64: "<f8"}[dtype]
    return torch.as_tensor(_DevView(ptr, shape, typestr), device=f"cuda:{device}")


def configure_from_workload(ctx: Context, w, pos_stride=4, frc_stride=4, with_method=True):
    """Translate a neutral ``workloads.Workload`` description into psg setup calls (marshalling only).
    For metadynamics the hill store is left empty; the caller loads or deposits hills."""
    ctx.set_layout(w.R, w.N, 0 if w.shared_array else w.N, pos_stride, frc_stride)
    cvs = [{"type": _KIND[cv["kind"]], "groups": cv["groups"], "axis": cv["axis"], "period": cv["period"]}
           for cv in w.cvs]
    ctx.set_cvs(cvs, w.slot_atom, None, w.atom_weight)
    if not with_method:
        return
    p = w.params
    if w.method == "harmonic":
        ctx.set_harmonic(p["kspring"], p["centers"])
    elif w.method == "metad":
        ctx.set_metad(p["sigma"], p["w0"], p["kB_deltaT"], p["capacity"], p["stride"])
    elif w.method == "abf":
        ctx.set_abf(p["lower"], p["upper"], p["shape"], p["periodic"], p["n_threshold"])
