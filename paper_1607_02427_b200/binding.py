"""Thin ctypes binding of libdem_b200 (include/dem.h): argument marshalling only.

Every step of the path runs in the library's CUDA kernels; PyTorch is used for device memory and streams.  The
function names are the C ABI's.  There is NO CPU fallback: if libdem_b200.so is missing or cannot be loaded the import
of this module's `lib()` raises, and every call that computes needs CUDA tensors.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

DEM_OK, DEM_EINVAL, DEM_ENOMEM, DEM_ECUDA, DEM_EBOX, DEM_ERCUT, DEM_EOVERFLOW, DEM_ESTALE = 0, -1, -2, -3, -4, -5, -6, -7
DEM_F32, DEM_F64 = 0, 1
STATUS_NAMES = {0: "DEM_OK", -1: "DEM_EINVAL", -2: "DEM_ENOMEM", -3: "DEM_ECUDA", -4: "DEM_EBOX", -5: "DEM_ERCUT",
                -6: "DEM_EOVERFLOW", -7: "DEM_ESTALE"}

# every symbol include/dem.h declares (tests check that the built library exports all of them)
EXPORTS = ["dem_create", "dem_destroy", "dem_last_error", "dem_set_eps_par", "dem_create_shape", "dem_build_neighbors",
           "dem_get_neighbors", "dem_copy_neighbors", "dem_compute", "dem_get_counters", "dem_step", "dem_step_nvt", "dem_step_npt",
           "dem_energy", "dem_energy_static",
           "dem_compute_host", "dem_step_host", "dem_set_slices", "dem_set_pair_kernel", "dem_set_culling", "dem_version"]
# include/dem_bench.h (measurement hooks)
EXPORTS_BENCH = ["dem_set_l2_flush", "dem_set_timing", "dem_kernel_times", "dem_swept_totals", "dem_launch_count",
                 "dem_fp32_peak"]

_lib = None


class DemError(RuntimeError):
    def __init__(self, code, text):
        super().__init__("%s: %s" % (STATUS_NAMES.get(code, code), text))
        self.code = code


def lib():
    """Load libdem_b200.so (built in-tree by build.py).  A library that is missing or was built from other sources than
    the ones in the tree is rebuilt first; if that is impossible the call fails loudly (there is no CPU fallback)."""
    global _lib
    if _lib is None:
        path = _build.LIB
        if _build.stale():
            try:
                _build.build()
            except Exception as e:  # no nvcc, compile error: never fall back to anything else
                raise ImportError("libdem_b200.so is missing or older than its sources and could not be rebuilt (%s); "
                                  "there is no CPU fallback" % e)
        _lib = C.CDLL(path)
        _lib.dem_last_error.restype = C.c_char_p
        _lib.dem_version.restype = C.c_char_p
        _lib.dem_launch_count.restype = C.c_int64
        want = _build.source_hash()
        if want not in _lib.dem_version().decode():
            raise ImportError("libdem_b200.so reports '%s' but the sources hash to %s: rebuild with "
                              "`python -m paper_1607_02427_b200.build`" % (_lib.dem_version().decode(), want))
    return _lib


def _check(ctx, rc):
    if rc != DEM_OK:
        msg = lib().dem_last_error(ctx).decode() if ctx else ""
        raise DemError(rc, msg)


def _dev(t, dtype=None, name="tensor"):
    """Device pointer of a contiguous CUDA tensor (None -> NULL)."""
    if t is None:
        return C.c_void_p(0)
    if not t.is_cuda:
        raise TypeError("%s must be a CUDA tensor (there is no CPU path)" % name)
    if not t.is_contiguous():
        raise TypeError("%s must be contiguous" % name)
    if dtype is not None and t.dtype != dtype:
        raise TypeError("%s must have dtype %s, got %s" % (name, dtype, t.dtype))
    return C.c_void_p(t.data_ptr())


def _host(a):
    return C.c_void_p(0) if a is None else a.ctypes.data_as(C.c_void_p)


def _box(box):
    b = np.ascontiguousarray(box, dtype=np.float64)
    if b.shape != (3,):
        raise ValueError("box must have 3 entries")
    return b


class Dem:
    """One library context.  Methods are the C calls of include/dem.h with torch tensors for device arrays."""

    def __init__(self, dim, epsilon=1.0, precision="f32", stream=None):
        import torch

        self.torch = torch
        self.dim = dim
        self.precision = DEM_F64 if precision in ("f64", DEM_F64) else DEM_F32
        self.dtype = torch.float64 if self.precision == DEM_F64 else torch.float32
        self.np_dtype = np.float64 if self.precision == DEM_F64 else np.float32
        if stream is None and torch.cuda.is_available():
            stream = torch.cuda.current_stream().cuda_stream
        self._ctx = C.c_void_p()
        rc = lib().dem_create(C.byref(self._ctx), C.c_int(dim), C.c_double(epsilon), C.c_int(self.precision),
                              C.c_void_p(stream or 0))
        if rc != DEM_OK:
            raise DemError(rc, "dem_create failed")
        self.shapes = []
        self._n_last = 0

    def close(self):
        if self._ctx:
            lib().dem_destroy(self._ctx)
            self._ctx = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- dem_set_* -------------------------------------------------------------------------------------------
    def set_eps_par(self, eps_par):
        _check(self._ctx, lib().dem_set_eps_par(self._ctx, C.c_double(eps_par)))

    def set_slices(self, slices):
        _check(self._ctx, lib().dem_set_slices(self._ctx, C.c_int(slices)))

    def set_pair_kernel(self, which):
        """0 = packed search kernel, 1 = generic fused kernel, 2 = auto (default: search in 3D, generic in 2D)."""
        _check(self._ctx, lib().dem_set_pair_kernel(self._ctx, C.c_int(which)))

    def swept_totals(self):
        out = (C.c_int64 * 3)()
        _check(self._ctx, lib().dem_swept_totals(self._ctx, out))
        return dict(ee_swept=out[0], vf_swept=out[1], face_edges_swept=out[2])

    def set_culling(self, enabled):
        _check(self._ctx, lib().dem_set_culling(self._ctx, C.c_int(1 if enabled else 0)))

    def set_l2_flush(self, nbytes):
        _check(self._ctx, lib().dem_set_l2_flush(self._ctx, C.c_int64(nbytes)))

    def set_timing(self, level):
        """0 off, 1 pose + pair kernels, 2 every kernel of a step (include/dem_bench.h)."""
        _check(self._ctx, lib().dem_set_timing(self._ctx, C.c_int(int(level))))

    # ---- dem_create_shape ----------------------------------------------------------------------------------------
    def create_shape(self, verts, faces=(), edges=None, rounding=0.1, mass=1.0, inertia=(1.0, 1.0, 1.0)):
        v = np.ascontiguousarray(verts, dtype=np.float64).reshape(-1, 3)
        fo, fv = [0], []
        for f in faces:
            fv += [int(k) for k in f]
            fo.append(len(fv))
        fo = np.array(fo, dtype=np.int32)
        fv = np.array(fv if fv else [0], dtype=np.int32)
        e = None if edges is None else np.ascontiguousarray(edges, dtype=np.int32).reshape(-1, 2)
        inert = np.ascontiguousarray(inertia, dtype=np.float64)
        sid = C.c_int(-1)
        rc = lib().dem_create_shape(self._ctx, _host(v), C.c_int(len(v)), _host(fo) if len(faces) else C.c_void_p(0),
                                    _host(fv) if len(faces) else C.c_void_p(0), C.c_int(len(faces)), _host(e),
                                    C.c_int(0 if e is None else len(e)), C.c_double(rounding), C.c_double(mass),
                                    _host(inert), C.byref(sid))
        _check(self._ctx, rc)
        self.shapes.append(sid.value)
        return sid.value

    def create_shape_dict(self, s):
        """A shape dict of dem_inputs.py."""
        return self.create_shape(s["verts"], s["faces"], s["edges"], s["rounding"], s["mass"], s["inertia"])

    # ---- dem_build_neighbors / dem_get_neighbors -------------------------------------------------------------------
    def build_neighbors(self, pos, shape_id, box, r_cut):
        torch = self.torch
        n = pos.shape[0]
        rc = lib().dem_build_neighbors(self._ctx, _dev(pos, self.dtype, "pos"), _dev(shape_id, torch.int32, "shape_id"),
                                       C.c_int(n), _host(_box(box)), C.c_double(r_cut))
        _check(self._ctx, rc)
        self._n_last = n

    def get_neighbors(self):
        """(counts int32[N], list int32[N, max_count]) as torch tensors (copies; unused entries are -1)."""
        torch = self.torch
        stride, mx = C.c_int(), C.c_int()
        cp, lp = C.c_void_p(), C.c_void_p()
        _check(self._ctx, lib().dem_get_neighbors(self._ctx, C.byref(cp), C.byref(lp), C.byref(stride), C.byref(mx)))
        n = self._n_last
        width = max(mx.value, 1)
        counts = torch.empty(n, dtype=torch.int32, device="cuda")
        lst = torch.empty((n, width), dtype=torch.int32, device="cuda")
        _check(self._ctx, lib().dem_copy_neighbors(self._ctx, _dev(counts), _dev(lst), C.c_int(width)))
        torch.cuda.current_stream().synchronize()
        return counts, lst

    # ---- dem_compute -------------------------------------------------------------------------------------------------
    def compute(self, pos, quat, shape_id, virial=True, out=None):
        torch = self.torch
        n = pos.shape[0]
        if out is None:
            f = torch.empty((n, 4), dtype=self.dtype, device=pos.device)
            t = torch.empty((n, 4), dtype=self.dtype, device=pos.device)
            w = torch.empty((n, 6), dtype=self.dtype, device=pos.device) if virial else None
        else:
            f, t, w = out
        rc = lib().dem_compute(self._ctx, _dev(pos, self.dtype, "pos"), _dev(quat, self.dtype, "quat"),
                               _dev(shape_id, torch.int32, "shape_id"), C.c_int(n), _dev(f, self.dtype), _dev(t, self.dtype),
                               _dev(w, self.dtype) if w is not None else C.c_void_p(0))
        _check(self._ctx, rc)
        return f, t, w

    def get_counters(self):
        out = (C.c_int64 * 9)()
        _check(self._ctx, lib().dem_get_counters(self._ctx, out))
        return dict(pairs_evaluated=out[0], terms=out[1], active=out[2], degenerate=out[3], parallel=out[4],
                    pairs_listed=out[5], terms_swept=out[6], ee_swept=out[7], face_edges_swept=out[8])

    # ---- dem_step / dem_energy -----------------------------------------------------------------------------------------
    def step(self, pos, quat, vel, angmom, shape_id, box, dt, nsteps, skin, force=None, torque=None):
        torch = self.torch
        n = pos.shape[0]
        rc = lib().dem_step(self._ctx, _dev(pos, self.dtype, "pos"), _dev(quat, self.dtype, "quat"),
                            _dev(vel, self.dtype, "vel"), _dev(angmom, self.dtype, "angmom"),
                            _dev(shape_id, torch.int32, "shape_id"), C.c_int(n), _host(_box(box)), C.c_double(dt),
                            C.c_int(nsteps), C.c_double(skin), _dev(force, self.dtype), _dev(torque, self.dtype))
        _check(self._ctx, rc)
        self._n_last = n

    def step_nvt(self, pos, quat, vel, angmom, shape_id, box, dt, nsteps, skin, kT, tau, thermostat=(0.0, 0.0),
                 force=None, torque=None):
        """dem_step_nvt; returns ((xi, eta), g)."""
        torch = self.torch
        n = pos.shape[0]
        th = (C.c_double * 2)(float(thermostat[0]), float(thermostat[1]))
        dof = C.c_double(0.0)
        rc = lib().dem_step_nvt(self._ctx, _dev(pos, self.dtype, "pos"), _dev(quat, self.dtype, "quat"),
                                _dev(vel, self.dtype, "vel"), _dev(angmom, self.dtype, "angmom"),
                                _dev(shape_id, torch.int32, "shape_id"), C.c_int(n), _host(_box(box)), C.c_double(dt),
                                C.c_int(nsteps), C.c_double(skin), C.c_double(kT), C.c_double(tau), th, C.byref(dof),
                                _dev(force, self.dtype), _dev(torque, self.dtype))
        _check(self._ctx, rc)
        self._n_last = n
        return (th[0], th[1]), dof.value

    def step_npt(self, pos, quat, vel, angmom, shape_id, box, dt, nsteps, skin, kT, tau, pressure, tau_p,
                 state=(0.0, 0.0, 0.0), force=None, torque=None):
        """dem_step_npt; returns (box, (xi, eta, nu), g)."""
        torch = self.torch
        n = pos.shape[0]
        st = (C.c_double * 3)(*[float(x) for x in state])
        b = (C.c_double * 3)(*[float(x) for x in _box(box)])
        dof = C.c_double(0.0)
        rc = lib().dem_step_npt(self._ctx, _dev(pos, self.dtype, "pos"), _dev(quat, self.dtype, "quat"),
                                _dev(vel, self.dtype, "vel"), _dev(angmom, self.dtype, "angmom"),
                                _dev(shape_id, torch.int32, "shape_id"), C.c_int(n), b, C.c_double(dt), C.c_int(nsteps),
                                C.c_double(skin), C.c_double(kT), C.c_double(tau), C.c_double(pressure),
                                C.c_double(tau_p), st, C.byref(dof), _dev(force, self.dtype), _dev(torque, self.dtype))
        _check(self._ctx, rc)
        self._n_last = n
        return np.array(b[:]), (st[0], st[1], st[2]), dof.value

    def energy(self, quat, vel, angmom, shape_id, force):
        torch = self.torch
        out = (C.c_double * 3)()
        rc = lib().dem_energy(self._ctx, _dev(quat, self.dtype), _dev(vel, self.dtype), _dev(angmom, self.dtype),
                              _dev(shape_id, torch.int32), _dev(force, self.dtype), C.c_int(quat.shape[0]), out)
        _check(self._ctx, rc)
        return np.array(out[:])

    def energy_static(self, quat, vel, angmom, shape_id, force, out):
        """dem_energy_static: `out` is a DEVICE float64 tensor of 3 entries; asynchronous, allocates nothing."""
        torch = self.torch
        rc = lib().dem_energy_static(self._ctx, _dev(quat, self.dtype), _dev(vel, self.dtype), _dev(angmom, self.dtype),
                                     _dev(shape_id, torch.int32), _dev(force, self.dtype), C.c_int(quat.shape[0]),
                                     _dev(out, torch.float64))
        _check(self._ctx, rc)

    # ---- host-buffer forms ---------------------------------------------------------------------------------------------
    def _hostarr(self, a, name, width=4):
        """numpy array or CPU torch tensor (pinned or not) -> (pointer, keepalive)."""
        if a is None:
            return C.c_void_p(0), None
        if hasattr(a, "data_ptr"):
            if a.is_cuda:
                raise TypeError("%s must be a HOST buffer for the *_host calls" % name)
            return C.c_void_p(a.data_ptr()), a
        return a.ctypes.data_as(C.c_void_p), a

    def compute_host(self, pos, quat, shape_id, box, r_cut, force, torque, virial=None):
        n = pos.shape[0]
        p = [self._hostarr(x, nm) for x, nm in ((pos, "pos"), (quat, "quat"), (shape_id, "shape_id"),
                                                 (force, "force"), (torque, "torque"), (virial, "virial"))]
        rc = lib().dem_compute_host(self._ctx, p[0][0], p[1][0], p[2][0], C.c_int(n), _host(_box(box)),
                                    C.c_double(r_cut), p[3][0], p[4][0], p[5][0])
        _check(self._ctx, rc)

    def step_host(self, pos, quat, vel, angmom, shape_id, box, dt, nsteps, skin, force=None, torque=None):
        n = pos.shape[0]
        p = [self._hostarr(x, nm) for x, nm in ((pos, "pos"), (quat, "quat"), (vel, "vel"), (angmom, "angmom"),
                                                 (shape_id, "shape_id"), (force, "force"), (torque, "torque"))]
        rc = lib().dem_step_host(self._ctx, p[0][0], p[1][0], p[2][0], p[3][0], p[4][0], C.c_int(n),
                                 _host(_box(box)), C.c_double(dt), C.c_int(nsteps), C.c_double(skin), p[5][0], p[6][0])
        _check(self._ctx, rc)

    # ---- accounting ------------------------------------------------------------------------------------------------------
    KERNEL_KINDS = ("pose", "pair", "reduce", "kick_drift", "neigh", "build", "flush", "other")

    def kernel_times(self):
        """dem_kernel_times: {kind: (launches, ms)} since the last call."""
        n, ms = (C.c_int64 * 8)(), (C.c_double * 8)()
        _check(self._ctx, lib().dem_kernel_times(self._ctx, n, ms))
        return {k: (n[i], ms[i]) for i, k in enumerate(self.KERNEL_KINDS)}

    def launch_count(self):
        return int(lib().dem_launch_count(self._ctx))

    def fp32_peak(self, iters=1 << 16):
        tf = C.c_double()
        _check(self._ctx, lib().dem_fp32_peak(self._ctx, C.c_int(iters), C.byref(tf)))
        return tf.value


def from_state(state, precision=None, device="cuda"):
    """Context + device tensors for a state dict of dem_inputs.py.  Returns (Dem, dict of tensors)."""
    import torch

    precision = precision or state.get("dtype", "f32")
    d = Dem(state["dim"], state.get("epsilon", 1.0), precision)
    for s in state["shapes"]:
        d.create_shape_dict(s)
    t = {}
    for k in ("pos", "quat", "vel", "angmom"):
        t[k] = torch.tensor(np.ascontiguousarray(state[k], dtype=d.np_dtype), device=device)
    t["shape_id"] = torch.tensor(np.ascontiguousarray(state["shape_id"], dtype=np.int32), device=device)
    return d, t
