"""ctypes wrapper around the CPU oracle (oracle/sph_oracle.c).

TEST INFRASTRUCTURE: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this package.  It never imports the CUDA binding.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import build as _build


class OrcParams(C.Structure):
    _fields_ = [
        ("dim", C.c_int),
        ("dp", C.c_double), ("h", C.c_double), ("rho0", C.c_double), ("c0", C.c_double),
        ("gamma", C.c_double), ("alpha", C.c_double), ("delta", C.c_double),
        ("g", C.c_double * 3),
        ("cfl", C.c_double),
        ("domain_min", C.c_double * 3), ("domain_max", C.c_double * 3),
        ("periodic", C.c_int * 3),
        ("eta2_coef", C.c_double),
        ("ddt_over_boundary", C.c_int),
        ("rho_bound_floor", C.c_int),
        ("cell_div", C.c_int),
        ("cell_size", C.c_double),
        ("visco_model", C.c_int),
        ("nu0", C.c_double),
        ("ddt_model", C.c_int),
        ("boundary_model", C.c_int),
        ("mdbc_slip", C.c_int),
        ("mdbc_det_min", C.c_double),
        ("shift_model", C.c_int),
        ("shift_coef", C.c_double),
        ("shift_fs_conc", C.c_double),
        ("shift_alpha_n", C.c_double),
        ("shift_beta_n", C.c_double),
    ]


class OrcMotion(C.Structure):
    _fields_ = [("group", C.c_int), ("axis", C.c_int), ("stroke", C.c_double),
                ("period", C.c_double), ("phase", C.c_double)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        L.orc_alphaD.restype = C.c_double
        L.orc_alphaD.argtypes = [C.c_int, C.c_double]
        L.orc_W.restype = C.c_double
        L.orc_W.argtypes = [C.c_int, C.c_double, C.c_double]
        L.orc_fab.restype = C.c_double
        L.orc_fab.argtypes = [C.c_int, C.c_double, C.c_double]
        L.orc_eos.restype = C.c_double
        L.orc_eos.argtypes = [C.POINTER(OrcParams), C.c_double]
        L.orc_dt.restype = C.c_double
        L.orc_num_threads.restype = C.c_int
        _lib = L
    return _lib


def make_params(p: dict) -> OrcParams:
    s = OrcParams()
    for k in ("dim", "dp", "h", "rho0", "c0", "gamma", "alpha", "delta", "cfl", "eta2_coef",
              "ddt_over_boundary", "rho_bound_floor", "cell_div", "cell_size"):
        setattr(s, k, p[k])
    for k in ("g", "domain_min", "domain_max"):
        getattr(s, k)[:] = [float(x) for x in p[k]]
    s.periodic[:] = [int(x) for x in p["periodic"]]
    s.visco_model = int(p.get("visco_model", 0))
    s.nu0 = float(p.get("nu0", 0.0))
    s.ddt_model = int(p.get("ddt_model", 0))
    s.boundary_model = int(p.get("boundary_model", 0))
    s.mdbc_slip = int(p.get("mdbc_slip", 0))
    s.mdbc_det_min = float(p.get("mdbc_det_min", 1e-3))
    s.shift_model = int(p.get("shift_model", 0))
    s.shift_coef = float(p.get("shift_coef", 2.0))
    s.shift_fs_conc = float(p.get("shift_fs_conc", 0.0))
    s.shift_alpha_n = float(p.get("shift_alpha_n", 0.0))
    s.shift_beta_n = float(p.get("shift_beta_n", 0.0))
    return s


def _ptr(a, ct):
    return a.ctypes.data_as(C.POINTER(ct))


def W(dim, h, r):
    return lib().orc_W(dim, h, r)


def fab(dim, h, r):
    return lib().orc_fab(dim, h, r)


def alphaD(dim, h):
    return lib().orc_alphaD(dim, h)


def eos(p: dict, rho: float) -> float:
    sp = make_params(p)
    return lib().orc_eos(C.byref(sp), rho)


def grid(p: dict):
    sp = make_params(p)
    cs = C.c_double()
    nc = (C.c_int * 3)()
    r2u = C.c_float()
    lib().orc_grid(C.byref(sp), C.byref(cs), nc, C.byref(r2u))
    return cs.value, (nc[0], nc[1], nc[2]), np.float32(r2u.value)


def canonicalize(p: dict, pos: np.ndarray):
    """C1: positions (n,3) float64 -> cell (n,3) int32, u (n,3) float32, out (n,) uint8."""
    pos = np.ascontiguousarray(pos, np.float64)
    n = pos.shape[0]
    cell = np.zeros((n, 3), np.int32)
    u = np.zeros((n, 3), np.float32)
    out = np.zeros(n, np.uint8)
    sp = make_params(p)
    lib().orc_canonicalize(C.byref(sp), C.c_int64(n), _ptr(pos, C.c_double), _ptr(cell, C.c_int32),
                           _ptr(u, C.c_float), _ptr(out, C.c_uint8))
    return cell, u, out


def position(p: dict, cell: np.ndarray, u: np.ndarray) -> np.ndarray:
    n = cell.shape[0]
    pos = np.zeros((n, 3), np.float64)
    sp = make_params(p)
    lib().orc_position(C.byref(sp), C.c_int64(n), _ptr(cell, C.c_int32), _ptr(u, C.c_float),
                       _ptr(pos, C.c_double))
    return pos


def neighbour_list(p: dict, cell, u_unused, ptype, out):
    """C3: keys, stable permutation, cellstart (2*ncells + 2 entries)."""
    n = cell.shape[0]
    sp = make_params(p)
    key = np.zeros(n, np.uint32)
    ptype = np.ascontiguousarray(ptype, np.uint8)
    lib().orc_keys(C.byref(sp), C.c_int64(n), _ptr(cell, C.c_int32), _ptr(ptype, C.c_uint8),
                   _ptr(out, C.c_uint8), _ptr(key, C.c_uint32))
    _, nc, _ = grid(p)
    ncells = nc[0] * nc[1] * nc[2]
    nkeys = 2 * ncells + 1
    perm = np.zeros(n, np.uint32)
    cellstart = np.zeros(nkeys + 1, np.uint32)
    lib().orc_sort(C.c_int64(n), _ptr(key, C.c_uint32), C.c_uint32(nkeys), _ptr(perm, C.c_uint32),
                   _ptr(cellstart, C.c_uint32))
    return key, perm, cellstart


def interactions(p: dict, cell, u, out, vel, rho, ptype, mode: int = 1):
    """One interaction pass. Returns dict(acc (n,3) f64, drho (n,) f64, nbcount u32, viscmax,
    n_diff = #pairs where the fp32 predicate C2 and the exact double predicate disagree)."""
    n = cell.shape[0]
    vel = np.ascontiguousarray(vel, np.float64)
    rho = np.ascontiguousarray(rho, np.float64)
    ptype = np.ascontiguousarray(ptype, np.uint8)
    acc = np.zeros((n, 3), np.float64)
    drho = np.zeros(n, np.float64)
    nb = np.zeros(n, np.uint32)
    visc = C.c_double()
    ndiff = C.c_uint64()
    sp = make_params(p)
    rc = lib().orc_interactions(C.byref(sp), C.c_int64(n), _ptr(cell, C.c_int32), _ptr(u, C.c_float),
                                _ptr(out, C.c_uint8), _ptr(vel, C.c_double), _ptr(rho, C.c_double),
                                _ptr(ptype, C.c_uint8), C.c_int(mode), _ptr(acc, C.c_double),
                                _ptr(drho, C.c_double), _ptr(nb, C.c_uint32), C.byref(visc),
                                C.byref(ndiff))
    assert rc == 0
    return dict(acc=acc, drho=drho, nbcount=nb, viscmax=visc.value, n_diff=ndiff.value)


def mdbc(p: dict, cell, u, out, vel, rho, ptype, normals, vwall=None, mode: int = 1):
    """mDBC, Eq. 38-39: returns (vel, rho, status) with the boundary entries replaced."""
    n = cell.shape[0]
    vel = np.ascontiguousarray(vel, np.float64).copy()
    rho = np.ascontiguousarray(rho, np.float64).copy()
    ptype = np.ascontiguousarray(ptype, np.uint8)
    normals = np.ascontiguousarray(normals, np.float64)
    status = np.zeros(n, np.uint8)
    sp = make_params(p)
    vw = None if vwall is None else np.ascontiguousarray(vwall, np.float64)
    rc = lib().orc_mdbc(C.byref(sp), C.c_int64(n), _ptr(cell, C.c_int32), _ptr(u, C.c_float),
                        _ptr(out, C.c_uint8), _ptr(vel, C.c_double), _ptr(rho, C.c_double),
                        _ptr(ptype, C.c_uint8), _ptr(normals, C.c_double),
                        None if vw is None else _ptr(vw, C.c_double), C.c_int(mode), _ptr(status, C.c_uint8))
    assert rc == 0
    return vel, rho, status


def concentration(p: dict, cell, u, out, rho, ptype, mode: int = 1):
    """C_a = sum_b V_b W_ab over all particles, self included (Eq. 53)."""
    n = cell.shape[0]
    rho = np.ascontiguousarray(rho, np.float64)
    ptype = np.ascontiguousarray(ptype, np.uint8)
    conc = np.zeros(n, np.float64)
    sp = make_params(p)
    rc = lib().orc_concentration(C.byref(sp), C.c_int64(n), _ptr(cell, C.c_int32), _ptr(u, C.c_float),
                                 _ptr(out, C.c_uint8), _ptr(rho, C.c_double), _ptr(ptype, C.c_uint8),
                                 C.c_int(mode), _ptr(conc, C.c_double))
    assert rc == 0
    return conc


def shift_velocity(p: dict, cell, u, out, vel, rho, ptype, conc=None, mode: int = 1):
    """Shifting velocity delta r / dt (Eq. 40-41, 53-54) and grad C of every fluid particle."""
    n = cell.shape[0]
    vel = np.ascontiguousarray(vel, np.float64)
    rho = np.ascontiguousarray(rho, np.float64)
    ptype = np.ascontiguousarray(ptype, np.uint8)
    if conc is None:
        conc = concentration(p, cell, u, out, rho, ptype, mode)
    conc = np.ascontiguousarray(conc, np.float64)
    shift = np.zeros((n, 3), np.float64)
    gradc = np.zeros((n, 3), np.float64)
    sp = make_params(p)
    rc = lib().orc_shift_velocity(C.byref(sp), C.c_int64(n), _ptr(cell, C.c_int32), _ptr(u, C.c_float),
                                  _ptr(out, C.c_uint8), _ptr(vel, C.c_double), _ptr(rho, C.c_double),
                                  _ptr(ptype, C.c_uint8), _ptr(conc, C.c_double), C.c_int(mode),
                                  _ptr(shift, C.c_double), _ptr(gradc, C.c_double))
    assert rc == 0
    return shift, gradc


def dt(p: dict, acc, ptype, out, viscmax: float) -> float:
    n = acc.shape[0]
    sp = make_params(p)
    ptype = np.ascontiguousarray(ptype, np.uint8)
    f = lib().orc_dt
    f.argtypes = [C.POINTER(OrcParams), C.c_int64, C.POINTER(C.c_double), C.POINTER(C.c_uint8),
                  C.POINTER(C.c_uint8), C.c_double]
    return f(C.byref(sp), n, _ptr(acc, C.c_double), _ptr(ptype, C.c_uint8), _ptr(out, C.c_uint8),
             viscmax)


class State:
    """Oracle-side simulation state in the canonical form (C1)."""

    def __init__(self, p: dict, pos, vel, rho, ptype, motions=(), normals=None):
        self.p = dict(p)
        self.cell, self.u, self.out = canonicalize(p, pos)
        self.vel = np.ascontiguousarray(vel, np.float64).copy()
        self.rho = np.ascontiguousarray(rho, np.float64).copy()
        self.ptype = np.ascontiguousarray(ptype, np.uint8).copy()
        self.pos0 = position(p, self.cell, self.u)
        self.motions = list(motions)
        self.normals = None if normals is None else np.ascontiguousarray(normals, np.float64).copy()
        self.t = 0.0
        self.dt_hist = []

    @property
    def pos(self):
        return position(self.p, self.cell, self.u)

    def interactions(self, mode=1):
        return interactions(self.p, self.cell, self.u, self.out, self.vel, self.rho, self.ptype,
                            mode)

    def step(self, nsteps: int, mode: int = 1):
        n = self.cell.shape[0]
        sp = make_params(self.p)
        nm = len(self.motions)
        mot = (OrcMotion * max(nm, 1))()
        for i, m in enumerate(self.motions):
            mot[i].group, mot[i].axis = int(m["group"]), int(m["axis"])
            mot[i].stroke, mot[i].period, mot[i].phase = m["stroke"], m["period"], m["phase"]
        t = C.c_double(self.t)
        hist = np.zeros(nsteps, np.float64)
        rc = lib().orc_step(C.byref(sp), C.c_int64(n), _ptr(self.cell, C.c_int32),
                            _ptr(self.u, C.c_float), _ptr(self.out, C.c_uint8),
                            _ptr(self.vel, C.c_double), _ptr(self.rho, C.c_double),
                            _ptr(self.ptype, C.c_uint8), C.c_int(nsteps), mot, C.c_int(nm),
                            _ptr(self.pos0, C.c_double),
                            None if self.normals is None else _ptr(self.normals, C.c_double),
                            C.byref(t), _ptr(hist, C.c_double), C.c_int(mode))
        assert rc == 0
        self.t = t.value
        self.dt_hist.extend(hist.tolist())
        return self


    def step_verlet(self, nsteps: int, verlet_steps: int = 40, mode: int = 1):
        """Verlet scheme, Eq. 30-31 (one interaction pass per step); keeps the state n-1 and the step counter."""
        n = self.cell.shape[0]
        if not hasattr(self, "vel_m1"):
            self.vel_m1 = np.zeros_like(self.vel)
            self.rho_m1 = np.zeros_like(self.rho)
            self.kstep = 0
        sp = make_params(self.p)
        nm = len(self.motions)
        mot = (OrcMotion * max(nm, 1))()
        for i, m in enumerate(self.motions):
            mot[i].group, mot[i].axis = int(m["group"]), int(m["axis"])
            mot[i].stroke, mot[i].period, mot[i].phase = m["stroke"], m["period"], m["phase"]
        t = C.c_double(self.t)
        k = C.c_int64(self.kstep)
        hist = np.zeros(nsteps, np.float64)
        rc = lib().orc_step_verlet(C.byref(sp), C.c_int64(n), _ptr(self.cell, C.c_int32),
                                   _ptr(self.u, C.c_float), _ptr(self.out, C.c_uint8),
                                   _ptr(self.vel, C.c_double), _ptr(self.rho, C.c_double),
                                   _ptr(self.vel_m1, C.c_double), _ptr(self.rho_m1, C.c_double),
                                   _ptr(self.ptype, C.c_uint8), C.c_int(nsteps), C.c_int(verlet_steps),
                                   C.byref(k), mot, C.c_int(nm), _ptr(self.pos0, C.c_double),
                                   None if self.normals is None else _ptr(self.normals, C.c_double),
                                   C.byref(t), _ptr(hist, C.c_double), C.c_int(mode))
        assert rc == 0
        self.t = t.value
        self.kstep = k.value
        self.dt_hist.extend(hist.tolist())
        return self


def num_threads() -> int:
    return lib().orc_num_threads()


def set_num_threads(n: int) -> None:
    lib().orc_set_num_threads(C.c_int(n))
