"""Thin Python binding of libsph_b200.so (include/sph.h): argument marshalling only.

Every step of the path (cell keys, radix sort, cell ranges, reorder, particle interaction, dt
reduction, symplectic update) runs in the library's CUDA kernels.  PyTorch is used for device memory
(the allocator callbacks hand out torch.uint8 CUDA tensors) and for the stream.  There is no CPU
fallback: importing this module fails if the shared library is missing, and creating a context fails
without a CUDA device.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libsph_b200.so")

SPH_OK, SPH_E_BADARG, SPH_E_NOMEM, SPH_E_CUDA, SPH_E_STATE, SPH_E_OVERFLOW, SPH_E_NAN = 0, -1, -2, -3, -4, -5, -6
_ERRNAMES = {-1: "SPH_E_BADARG", -2: "SPH_E_NOMEM", -3: "SPH_E_CUDA", -4: "SPH_E_STATE",
             -5: "SPH_E_OVERFLOW", -6: "SPH_E_NAN"}

(SPH_POS, SPH_VEL, SPH_RHO, SPH_ACC, SPH_DRHODT, SPH_KEY, SPH_PERM, SPH_CELLSTART, SPH_NBCOUNT,
 SPH_CELL, SPH_OFFSET, SPH_PRESS, SPH_CONC, SPH_SHIFT) = range(1, 15)

ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p)
FREE_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)


class SphParams(C.Structure):
    _fields_ = [
        ("dim", C.c_int32),
        ("dp", C.c_double), ("h", C.c_double), ("rho0", C.c_double), ("c0", C.c_double),
        ("gamma", C.c_double), ("alpha", C.c_double), ("delta", C.c_double),
        ("g", C.c_double * 3),
        ("cfl", C.c_double),
        ("domain_min", C.c_double * 3), ("domain_max", C.c_double * 3),
        ("periodic", C.c_int32 * 3),
        ("eta2_coef", C.c_double),
        ("ddt_over_boundary", C.c_int32),
        ("rho_bound_floor", C.c_int32),
        ("cell_div", C.c_int32),
        ("cell_size", C.c_double),
        ("pi_kernel", C.c_int32),
        ("count_neighbours", C.c_int32),
        ("integrator", C.c_int32),
        ("verlet_steps", C.c_int32),
        ("visco_model", C.c_int32),
        ("ddt_model", C.c_int32),
        ("nu0", C.c_double),
        ("boundary_model", C.c_int32),
        ("mdbc_slip", C.c_int32),
        ("mdbc_det_min", C.c_double),
        ("shift_model", C.c_int32),
        ("shift_coef", C.c_double),
        ("shift_fs_conc", C.c_double),
        ("shift_alpha_n", C.c_double),
        ("shift_beta_n", C.c_double),
        ("compensated_sums", C.c_int32),
        ("dev_alloc", ALLOC_FN),
        ("dev_free", FREE_FN),
        ("user", C.c_void_p),
        ("cuda_stream", C.c_void_p),
    ]


class SphInfo(C.Structure):
    _fields_ = [
        ("n", C.c_int64), ("n_out", C.c_int64), ("n_bound", C.c_int64),
        ("ncell", C.c_int32 * 3), ("ncells", C.c_int64),
        ("cell_size", C.c_double), ("r2u", C.c_float),
        ("n_interactions", C.c_uint64), ("n_interactions_total", C.c_uint64),
        ("steps_done", C.c_int64), ("t", C.c_double), ("dt", C.c_double),
        ("pi_kernel", C.c_int32), ("device_flags", C.c_int32),
    ]


class SphTimings(C.Structure):
    _fields_ = [
        ("ms_key", C.c_double), ("ms_sort", C.c_double), ("ms_cellstart", C.c_double),
        ("ms_reorder", C.c_double), ("ms_interaction", C.c_double), ("ms_dt", C.c_double),
        ("ms_update", C.c_double),
        ("n_nl_builds", C.c_int64), ("n_interaction_passes", C.c_int64), ("n_kernel_launches", C.c_int64),
        ("ms_mdbc", C.c_double), ("ms_shift", C.c_double),
    ]


EXPORTS = ["sph_create", "sph_destroy", "sph_load_particles", "sph_set_motion", "sph_set_boundary_normals",
           "sph_compute_interactions", "sph_step", "sph_read_state", "sph_read_fields", "sph_get_info",
           "sph_set_profiling", "sph_get_timings", "sph_last_error", "sph_version", "sph_sort_keys_static"]
SPH_SORT_STATIC_MAX_N = 1 << 20


def _load():
    if not os.path.exists(_LIB_PATH):
        raise ImportError(
            f"{_LIB_PATH} is missing: build it with `python -m paper_2104_00537_b200.build` "
            "(there is no CPU fallback)")
    L = C.CDLL(_LIB_PATH)
    vp = C.c_void_p
    L.sph_create.argtypes = [C.POINTER(SphParams), C.POINTER(vp)]
    L.sph_destroy.argtypes = [vp]
    L.sph_destroy.restype = None
    L.sph_load_particles.argtypes = [vp, C.c_int64, vp, vp, vp, vp]
    L.sph_set_motion.argtypes = [vp, C.c_int32, C.c_int32, C.c_double, C.c_double, C.c_double]
    L.sph_set_boundary_normals.argtypes = [vp, vp]
    L.sph_compute_interactions.argtypes = [vp]
    L.sph_step.argtypes = [vp, C.c_int32]
    L.sph_read_state.argtypes = [vp, C.c_int32, vp, C.c_size_t]
    L.sph_read_fields.argtypes = [vp, C.c_int32, C.POINTER(C.c_int32), C.POINTER(C.c_void_p), C.POINTER(C.c_size_t)]
    L.sph_get_info.argtypes = [vp, C.POINTER(SphInfo)]
    L.sph_set_profiling.argtypes = [vp, C.c_int32]
    L.sph_get_timings.argtypes = [vp, C.POINTER(SphTimings)]
    L.sph_last_error.argtypes = [vp]
    L.sph_last_error.restype = C.c_char_p
    L.sph_version.restype = C.c_char_p
    L.sph_sort_keys_static.argtypes = [vp, C.c_int64, C.c_int32, vp, vp, vp, C.c_char_p, C.c_size_t]
    for name in EXPORTS:
        if name not in ("sph_destroy", "sph_last_error", "sph_version"):
            getattr(L, name).restype = C.c_int
    return L


lib = _load()


class SphError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"{_ERRNAMES.get(code, code)}: {msg}")
        self.code = code


def version() -> str:
    return lib.sph_version().decode()


def sort_keys_static(key_ptr, n, key_bits, key_sorted_ptr, perm_ptr, stream_ptr=None):
    """sph_sort_keys_static: the neighbour-list sort for callers that may not allocate device memory (a host code that
    owns all of HBM through its own pool, or a loop that cannot take the device-wide stall of cudaMalloc / cudaFree).
    The work space is a fixed array inside the library, so n <= SPH_SORT_STATIC_MAX_N.  All three pointers are raw
    DEVICE addresses of uint32[n] arrays on the current device (e.g. tensor.data_ptr()); stream_ptr is a cudaStream_t
    value (None = legacy default stream).  Only enqueues work.  The first call on a device does a one-off address look-up
    and belongs in set-up code; calls that can overlap on the GPU share the work space and race (see include/sph.h)."""
    msg = C.create_string_buffer(512)
    rc = lib.sph_sort_keys_static(key_ptr, n, key_bits, key_sorted_ptr, perm_ptr, stream_ptr, msg, len(msg))
    if rc != SPH_OK:
        raise SphError(rc, msg.value.decode())


class Sph:
    """One simulation context.  Method names follow the C ABI (sph_<name>)."""

    def __init__(self, params: dict, pi_kernel: int = 0, count_neighbours: bool = False,
                 stream=None, use_torch_allocator: bool = True):
        import torch  # device memory + streams only

        if not torch.cuda.is_available():
            raise SphError(SPH_E_CUDA, "no CUDA device: libsph_b200 has no CPU fallback")
        self._torch = torch
        self._bufs = {}
        sp = SphParams()
        for k in ("dim", "dp", "h", "rho0", "c0", "gamma", "alpha", "delta", "cfl", "eta2_coef",
                  "ddt_over_boundary", "rho_bound_floor", "cell_div", "cell_size"):
            setattr(sp, k, params[k])
        for k in ("g", "domain_min", "domain_max"):
            getattr(sp, k)[:] = [float(x) for x in params[k]]
        sp.periodic[:] = [int(x) for x in params["periodic"]]
        sp.pi_kernel = int(params.get("pi_kernel", pi_kernel))
        sp.count_neighbours = int(bool(count_neighbours))
        sp.integrator = int(params.get("integrator", 0))
        sp.verlet_steps = int(params.get("verlet_steps", 0))
        sp.visco_model = int(params.get("visco_model", 0))
        sp.nu0 = float(params.get("nu0", 0.0))
        sp.ddt_model = int(params.get("ddt_model", 0))
        for k in ("boundary_model", "mdbc_slip", "shift_model", "compensated_sums"):
            setattr(sp, k, int(params.get(k, 0)))
        for k in ("mdbc_det_min", "shift_coef", "shift_fs_conc", "shift_alpha_n", "shift_beta_n"):
            setattr(sp, k, float(params.get(k, 0.0)))
        self._stream = stream if stream is not None else torch.cuda.current_stream()
        sp.cuda_stream = self._stream.cuda_stream

        if use_torch_allocator:
            def _alloc(nbytes, _user):
                try:
                    with torch.cuda.stream(self._stream):
                        t = torch.empty(max(int(nbytes), 16), dtype=torch.uint8, device="cuda")
                except Exception:  # out of memory -> NULL -> SPH_E_NOMEM
                    return None
                self._bufs[t.data_ptr()] = t
                return t.data_ptr()

            def _free(ptr, _user):
                self._bufs.pop(ptr, None)

            self._alloc_cb, self._free_cb = ALLOC_FN(_alloc), FREE_FN(_free)
            sp.dev_alloc, sp.dev_free = self._alloc_cb, self._free_cb
        self._params = sp
        self._h = C.c_void_p()
        rc = lib.sph_create(C.byref(sp), C.byref(self._h))
        if rc != SPH_OK:
            raise SphError(rc, "sph_create failed: " + lib.sph_last_error(None).decode())
        self.n = 0

    # -- helpers ---------------------------------------------------------------------------------
    def _ck(self, rc):
        if rc != SPH_OK:
            raise SphError(rc, lib.sph_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            lib.sph_destroy(self._h)
            self._h = C.c_void_p()
            self._bufs.clear()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    # -- the C ABI ---------------------------------------------------------------------------------
    def load_particles(self, pos, vel, rho, ptype):
        pos = np.ascontiguousarray(pos, np.float64)
        vel = np.ascontiguousarray(vel, np.float32)
        rho = np.ascontiguousarray(rho, np.float32)
        ptype = np.ascontiguousarray(ptype, np.uint8)
        n = pos.shape[0]
        assert pos.shape == (n, 3) and vel.shape == (n, 3) and rho.shape == (n,) and ptype.shape == (n,)
        self._ck(lib.sph_load_particles(self._h, n, pos.ctypes.data, vel.ctypes.data, rho.ctypes.data,
                                        ptype.ctypes.data))
        self.n = n

    def load_particles_ptr(self, n, pos_ptr, vel_ptr, rho_ptr, type_ptr):
        """Same call with raw host pointers (e.g. pinned torch tensors)."""
        self._ck(lib.sph_load_particles(self._h, n, pos_ptr, vel_ptr, rho_ptr, type_ptr))
        self.n = n

    def set_motion(self, group, axis, stroke, period, phase=0.0):
        self._ck(lib.sph_set_motion(self._h, group, axis, stroke, period, phase))

    def set_boundary_normals(self, normals):
        normals = np.ascontiguousarray(normals, np.float64)
        assert normals.shape == (self.n, 3)
        self._ck(lib.sph_set_boundary_normals(self._h, normals.ctypes.data))

    def compute_interactions(self):
        self._ck(lib.sph_compute_interactions(self._h))

    def step(self, nsteps=1):
        self._ck(lib.sph_step(self._h, nsteps))

    def read_state(self, field, out=None):
        info = None
        n = self.n
        shapes = {SPH_POS: ((n, 3), np.float64), SPH_VEL: ((n, 3), np.float32), SPH_RHO: ((n,), np.float32),
                  SPH_ACC: ((n, 3), np.float32), SPH_DRHODT: ((n,), np.float32), SPH_KEY: ((n,), np.uint32),
                  SPH_PERM: ((n,), np.uint32), SPH_NBCOUNT: ((n,), np.uint32), SPH_CELL: ((n, 3), np.int32),
                  SPH_OFFSET: ((n, 3), np.float32), SPH_PRESS: ((n,), np.float32),
                  SPH_CONC: ((n,), np.float32), SPH_SHIFT: ((n, 3), np.float32)}
        if field == SPH_CELLSTART:
            info = self.get_info()
            shape, dt = (2 * info.ncells + 2,), np.uint32
        else:
            shape, dt = shapes[field]
        if out is None:
            out = np.empty(shape, dt)
        self._ck(lib.sph_read_state(self._h, field, out.ctypes.data, out.nbytes))
        return out

    def read_state_ptr(self, field, ptr, nbytes):
        self._ck(lib.sph_read_state(self._h, field, ptr, nbytes))

    def read_fields_ptr(self, fields, ptrs, nbytes):
        """Several fields in one call (one synchronisation): host pointers and sizes per field."""
        k = len(fields)
        f = (C.c_int32 * k)(*fields)
        d = (C.c_void_p * k)(*ptrs)
        b = (C.c_size_t * k)(*nbytes)
        self._ck(lib.sph_read_fields(self._h, k, f, d, b))

    def get_info(self) -> SphInfo:
        info = SphInfo()
        self._ck(lib.sph_get_info(self._h, C.byref(info)))
        return info

    def set_profiling(self, on: bool):
        self._ck(lib.sph_set_profiling(self._h, int(on)))

    def get_timings(self) -> SphTimings:
        t = SphTimings()
        self._ck(lib.sph_get_timings(self._h, C.byref(t)))
        return t

    def load_case(self, case):
        self.load_particles(case.pos, case.vel, case.rho, case.ptype)
        for m in case.motions:
            self.set_motion(m["group"], m["axis"], m["stroke"], m["period"], m["phase"])
        if self._params.boundary_model == 1 and getattr(case, "normals", None) is not None:
            self.set_boundary_normals(case.normals)
