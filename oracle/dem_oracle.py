"""ctypes access to the FP64 CPU oracle (oracle/dem_oracle.c).  TEST INFRASTRUCTURE, NOT PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / `--impl reference` legs may import this module.
It imports nothing from paper_1607_02427_b200 (the CUDA path) and the CUDA path imports nothing from here.
Argument marshalling only -- all arithmetic is in dem_oracle.c.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "dem_oracle.c")
_LIB = os.path.join(_HERE, "libdem_oracle.so")
DEFAULT_EPS_PAR = 1e-6  # reading R5: parallel <=> |d1 x d2|^2 < eps_par |d1|^2 |d2|^2


def build(force=False):
    """Compile the oracle with gcc (-O2, no FMA contraction, no fast-math).  With DEM_ORACLE_SANITIZE=1 in the
    environment a second library is built with -fsanitize=address,undefined and used instead (run python with
    LD_PRELOAD=$(gcc -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0; profiles/r02_sanitizers.md)."""
    san = os.environ.get("DEM_ORACLE_SANITIZE") == "1"
    out = _LIB.replace(".so", "_san.so") if san else _LIB
    flags = (["-O1", "-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined"]
             if san else ["-O2"])
    if force or not os.path.exists(out) or os.path.getmtime(out) < os.path.getmtime(_SRC):
        tmp = out + ".tmp%d" % os.getpid()
        subprocess.check_call(["gcc"] + flags + ["-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", _SRC, "-o", tmp, "-lm"])
        os.replace(tmp, out)
    return out


class _Shapes(C.Structure):
    _fields_ = [("nshapes", C.c_int), ("vert_off", C.c_void_p), ("verts", C.c_void_p), ("edge_off", C.c_void_p),
                ("edges", C.c_void_p), ("face_off", C.c_void_p), ("face_ptr", C.c_void_p), ("face_verts", C.c_void_p),
                ("rounding", C.c_void_p)]


class Term(C.Structure):
    _fields_ = [("type", C.c_int), ("k", C.c_int), ("l", C.c_int), ("branch", C.c_int), ("r", C.c_double),
                ("ci", C.c_double * 3), ("cj", C.c_double * 3)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_point_segment.restype = C.c_double
        for name in ("orc_segment_segment", "orc_point_polygon", "orc_pair_terms", "orc_neighbors", "orc_compute",
                     "orc_compute_cells", "orc_step", "orc_num_threads"):
            getattr(_lib, name).restype = C.c_int
        _lib.orc_wca.restype = None
        _lib.orc_energy.restype = None
        _lib.orc_set_num_threads.restype = None
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _f64(a, shape=None):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a if shape is None else a.reshape(shape)


class ShapeTable:
    """Flat arrays describing a list of shape dicts (see dem_inputs.py) in the layout of `orc_shapes`."""

    def __init__(self, shapes):
        self.shapes = shapes
        self.vert_off = np.cumsum([0] + [len(s["verts"]) for s in shapes]).astype(np.int32)
        self.verts = _f64(np.concatenate([np.asarray(s["verts"], dtype=np.float64).reshape(-1, 3) for s in shapes]))
        self.edge_off = np.cumsum([0] + [len(s["edges"]) for s in shapes]).astype(np.int32)
        self.edges = np.ascontiguousarray(
            np.concatenate([np.asarray(s["edges"], dtype=np.int32).reshape(-1, 2) for s in shapes]), dtype=np.int32)
        self.face_off = np.cumsum([0] + [len(s["faces"]) for s in shapes]).astype(np.int32)
        ptr, fv = [0], []
        for s in shapes:
            for f in s["faces"]:
                fv += list(f)
                ptr.append(len(fv))
        self.face_ptr = np.array(ptr, dtype=np.int32)
        self.face_verts = np.array(fv if fv else [0], dtype=np.int32)
        self.rounding = _f64([s["rounding"] for s in shapes])
        self.mass = _f64([s["mass"] for s in shapes])
        self.inertia = _f64(np.stack([s["inertia"] for s in shapes]))
        self.c = _Shapes(len(shapes), _p(self.vert_off), _p(self.verts), _p(self.edge_off), _p(self.edges),
                         _p(self.face_off), _p(self.face_ptr), _p(self.face_verts), _p(self.rounding))


# ---- primitives ------------------------------------------------------------------------------------------------
def point_segment(p, a, b):
    c = np.zeros(3)
    t = lib().orc_point_segment(_p(_f64(p)), _p(_f64(a)), _p(_f64(b)), _p(c))
    return c, t


def segment_segment(p1, q1, p2, q2, eps_par=DEFAULT_EPS_PAR):
    c1, c2 = np.zeros(3), np.zeros(3)
    br = lib().orc_segment_segment(_p(_f64(p1)), _p(_f64(q1)), _p(_f64(p2)), _p(_f64(q2)), C.c_double(eps_par),
                                   _p(c1), _p(c2))
    return c1, c2, br


def point_polygon(p, poly):
    poly = _f64(poly).reshape(-1, 3)
    c = np.zeros(3)
    inside = lib().orc_point_polygon(_p(_f64(p)), _p(poly), C.c_int(len(poly)), _p(c))
    return c, inside


def wca(r, sigma, eps=1.0):
    u, f = C.c_double(), C.c_double()
    lib().orc_wca(C.c_double(r), C.c_double(sigma), C.c_double(eps), C.byref(u), C.byref(f))
    return u.value, f.value


# ---- pair / system level ---------------------------------------------------------------------------------------
def pair_terms(shapes, si, sj, qi, qj, d, eps=1.0, eps_par=DEFAULT_EPS_PAR, dim=None):
    """All Eq. 1 / Eq. 2 terms of the ordered pair (i, j) with d = x_j - x_i.  Returns (list of dict, sums dict)."""
    tab = shapes if isinstance(shapes, ShapeTable) else ShapeTable(shapes)
    dim = tab.shapes[si]["dim"] if dim is None else dim
    cap = 1 << 16
    buf = (Term * cap)()
    out = np.zeros(17)
    n = lib().orc_pair_terms(C.byref(tab.c), C.c_int(dim), C.c_int(si), C.c_int(sj), _p(_f64(qi)), _p(_f64(qj)),
                             _p(_f64(d)), C.c_double(eps), C.c_double(eps_par), buf, C.c_int(cap), _p(out))
    assert n <= cap
    terms = [dict(type=t.type, k=t.k, l=t.l, branch=t.branch, r=t.r, ci=np.array(t.ci[:]), cj=np.array(t.cj[:]))
             for t in buf[:n]]
    sums = dict(Fi=out[0:3].copy(), Ti=out[3:6].copy(), Tj=out[6:9].copy(), u=out[9], W=out[10:16].copy(), rmin=out[16])
    return terms, sums


def neighbors(state, r_cut=None, subset=None, stride=64):
    """Neighbour rows by definition O1.  Returns (counts, list[rows, stride]) with each row sorted by j."""
    pos = _f64(state["pos"])
    n = len(pos)
    sub = None if subset is None else np.ascontiguousarray(subset, dtype=np.int32)
    rows = n if sub is None else len(sub)
    r_cut = state["r_cut"] if r_cut is None else r_cut
    while True:
        counts = np.zeros(rows, dtype=np.int32)
        lst = np.full((rows, stride), -1, dtype=np.int32)
        mx = lib().orc_neighbors(C.c_int(state["dim"]), C.c_int(n), _p(_f64(state["box"])), _p(pos),
                                 C.c_double(r_cut), _p(sub), C.c_int(rows), _p(counts), _p(lst), C.c_int(stride))
        if mx <= stride:
            return counts, lst
        stride = mx


def _check_min_image(state, tab):
    """The all-pairs minimum-image sum equals the periodic sum only if no interaction reaches beyond half a box
    edge (reading R9): reach = max (R_i + R_j + 2^(1/6) (rho_i + rho_j))."""
    rad = [np.sqrt((np.asarray(s["verts"]) ** 2).sum(1).max()) for s in tab.shapes]
    reach = max(a + b + 2 ** (1 / 6) * (sa["rounding"] + sb["rounding"])
                for a, sa in zip(rad, tab.shapes) for b, sb in zip(rad, tab.shapes))
    box = np.asarray(state["box"], dtype=np.float64)
    if np.any(box[:state["dim"]] < 2 * reach):
        raise ValueError("box edge %s < 2 x interaction reach %g: minimum image invalid" % (box, reach))


def compute(state, subset=None, use_reject=True, eps_par=DEFAULT_EPS_PAR, pos=None, quat=None, cells=False):
    """Per-particle force+energy (rows,4), torque (rows,4), virial (rows,6), counters(5) by the definition.
    cells=True: orc_compute_cells, the same sums over the same pairs in the same order (bit-identical to the all-pairs
    loop with the exact reject), found through a plain cell grid instead of an O(N) scan per particle."""
    tab = state.get("_tab") or ShapeTable(state["shapes"])
    pos = _f64(state["pos"] if pos is None else pos)
    quat = _f64(state["quat"] if quat is None else quat)
    n = len(pos)
    _check_min_image(state, tab)
    sub = None if subset is None else np.ascontiguousarray(subset, dtype=np.int32)
    rows = n if sub is None else len(sub)
    f, t, w = np.zeros((rows, 4)), np.zeros((rows, 4)), np.zeros((rows, 6))
    cnt = np.zeros(5, dtype=np.int64)
    sid = np.ascontiguousarray(state["shape_id"], dtype=np.int32)
    if cells:
        if not use_reject:
            raise ValueError("the cell grid only finds pairs inside the interaction reach: use_reject must stay on")
        lib().orc_compute_cells(C.byref(tab.c), C.c_int(state["dim"]), C.c_int(n), _p(_f64(state["box"])), _p(pos),
                                _p(quat), _p(sid), C.c_double(state["epsilon"]), C.c_double(eps_par), _p(sub),
                                C.c_int(rows), _p(f), _p(t), _p(w), _p(cnt))
        return f, t, w, cnt
    lib().orc_compute(C.byref(tab.c), C.c_int(state["dim"]), C.c_int(n), _p(_f64(state["box"])), _p(pos), _p(quat),
                      _p(sid), C.c_double(state["epsilon"]), C.c_double(eps_par), C.c_int(1 if use_reject else 0),
                      _p(sub), C.c_int(rows), _p(f), _p(t), _p(w), _p(cnt))
    return f, t, w, cnt


def step(state, dt, nsteps, eps_par=DEFAULT_EPS_PAR, record_energy=True):
    """NVE integration of a COPY of the state.  Returns dict(pos, quat, vel, angmom, force, torque, energies)."""
    tab = state.get("_tab") or ShapeTable(state["shapes"])
    pos, quat = _f64(state["pos"]).copy(), _f64(state["quat"]).copy()
    vel, ang = _f64(state["vel"]).copy(), _f64(state["angmom"]).copy()
    n = len(pos)
    f, t = np.zeros((n, 4)), np.zeros((n, 4))
    en = np.zeros((nsteps + 1, 3)) if record_energy else None
    sid = np.ascontiguousarray(state["shape_id"], dtype=np.int32)
    lib().orc_step(C.byref(tab.c), _p(tab.mass), _p(tab.inertia), C.c_int(state["dim"]), C.c_int(n),
                   _p(_f64(state["box"])), _p(pos), _p(quat), _p(vel), _p(ang), _p(sid), C.c_double(state["epsilon"]),
                   C.c_double(eps_par), C.c_double(dt), C.c_int(nsteps), _p(f), _p(t), _p(en))
    return dict(pos=pos, quat=quat, vel=vel, angmom=ang, force=f, torque=t, energies=en)


def step_nvt(state, dt, nsteps, kT, tau, thermo=(0.0, 0.0), eps_par=DEFAULT_EPS_PAR):
    """Nose-Hoover NVT integration of a COPY of the state (orc_step_nvt; R19).  Returns dict(pos, quat, vel,
    angmom, force, torque, energies [nsteps+1][5] = U, K_trans, K_rot, xi, eta, thermo = final (xi, eta), dof = g)."""
    tab = state.get("_tab") or ShapeTable(state["shapes"])
    pos, quat = _f64(state["pos"]).copy(), _f64(state["quat"]).copy()
    vel, ang = _f64(state["vel"]).copy(), _f64(state["angmom"]).copy()
    n = len(pos)
    f, t = np.zeros((n, 4)), np.zeros((n, 4))
    en = np.zeros((nsteps + 1, 5))
    th = np.array(thermo, dtype=np.float64)
    sid = np.ascontiguousarray(state["shape_id"], dtype=np.int32)
    fn = lib().orc_step_nvt
    fn.restype = C.c_double
    g = fn(C.byref(tab.c), _p(tab.mass), _p(tab.inertia), C.c_int(state["dim"]), C.c_int(n), _p(_f64(state["box"])),
           _p(pos), _p(quat), _p(vel), _p(ang), _p(sid), C.c_double(state["epsilon"]), C.c_double(eps_par),
           C.c_double(dt), C.c_int(nsteps), C.c_double(kT), C.c_double(tau), _p(th), _p(f), _p(t), _p(en))
    return dict(pos=pos, quat=quat, vel=vel, angmom=ang, force=f, torque=t, energies=en, thermo=th, dof=g)


def step_npt(state, dt, nsteps, kT, tau, pressure, tau_p, baro=(0.0, 0.0, 0.0), eps_par=DEFAULT_EPS_PAR):
    """Nose-Hoover + MTK NPT integration of a COPY of the state (orc_step_npt; R22).  Returns dict(pos, quat,
    vel, angmom, box, force, torque, energies [nsteps+1][8] = U, K_trans, K_rot, xi, eta, nu, V, tr W, baro = final
    (xi, eta, nu), dof = g)."""
    tab = state.get("_tab") or ShapeTable(state["shapes"])
    pos, quat = _f64(state["pos"]).copy(), _f64(state["quat"]).copy()
    vel, ang = _f64(state["vel"]).copy(), _f64(state["angmom"]).copy()
    box = _f64(state["box"]).copy()
    n = len(pos)
    f, t = np.zeros((n, 4)), np.zeros((n, 4))
    en = np.zeros((nsteps + 1, 8))
    b = np.array(baro, dtype=np.float64)
    sid = np.ascontiguousarray(state["shape_id"], dtype=np.int32)
    fn = lib().orc_step_npt
    fn.restype = C.c_double
    g = fn(C.byref(tab.c), _p(tab.mass), _p(tab.inertia), C.c_int(state["dim"]), C.c_int(n), _p(box), _p(pos), _p(quat),
           _p(vel), _p(ang), _p(sid), C.c_double(state["epsilon"]), C.c_double(eps_par), C.c_double(dt), C.c_int(nsteps),
           C.c_double(kT), C.c_double(tau), C.c_double(pressure), C.c_double(tau_p), _p(b), _p(f), _p(t), _p(en))
    return dict(pos=pos, quat=quat, vel=vel, angmom=ang, box=box, force=f, torque=t, energies=en, baro=b, dof=g)


def energy(state, force):
    tab = state.get("_tab") or ShapeTable(state["shapes"])
    out = np.zeros(3)
    sid = np.ascontiguousarray(state["shape_id"], dtype=np.int32)
    lib().orc_energy(C.c_int(state["dim"]), C.c_int(len(sid)), _p(tab.mass), _p(tab.inertia), _p(sid),
                     _p(_f64(state["quat"])), _p(_f64(state["vel"])), _p(_f64(state["angmom"])), _p(_f64(force)), _p(out))
    return out


def num_threads():
    return lib().orc_num_threads()


def set_num_threads(n):
    lib().orc_set_num_threads(C.c_int(n))
