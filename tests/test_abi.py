"""CPU-side checks of the C-ABI boundary: the library loads, exports every symbol include/sph.h
declares, validates parameters before touching the device, and fails loudly without a GPU."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def sph():
    from paper_2104_00537_b200 import build
    build.build()
    from paper_2104_00537_b200 import sph as mod
    return mod


def declared_functions():
    src = open(os.path.join(ROOT, "include", "sph.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(sph_[a-z_]+)\s*\(", src)))


def test_header_symbols_are_exported(sph):
    names = declared_functions()
    assert "sph_create" in names and "sph_step" in names and "sph_read_state" in names
    assert "sph_load_particles" in names and "sph_compute_interactions" in names
    raw = C.CDLL(os.path.join(ROOT, "paper_2104_00537_b200", "libsph_b200.so"))
    for n in names:
        assert hasattr(raw, n), f"{n} declared in include/sph.h but not exported"
    assert sorted(sph.EXPORTS) == names
    assert "sm_100a" in sph.version()


def _params(sph, **kw):
    p = sph.SphParams()
    p.dim, p.dp, p.h, p.rho0, p.c0, p.gamma = 3, 0.02, 0.0416, 1000.0, 17.0, 7.0
    p.alpha, p.delta, p.cfl, p.eta2_coef, p.cell_div = 0.01, 0.1, 0.2, 0.001, 1
    p.domain_min[:] = [0, 0, 0]
    p.domain_max[:] = [1, 1, 1]
    for k, v in kw.items():
        setattr(p, k, v)
    return p


@pytest.mark.parametrize("kw", [dict(dim=4), dict(dp=0.0), dict(h=-1.0), dict(cfl=0.0), dict(cell_div=0),
                                dict(cell_div=4), dict(cell_size=0.01), dict(gamma=0.0), dict(pi_kernel=7)])
def test_bad_parameters_are_rejected_before_device_use(sph, kw):
    h = C.c_void_p()
    rc = sph.lib.sph_create(C.byref(_params(sph, **kw)), C.byref(h))
    assert rc == sph.SPH_E_BADARG and not h.value


def test_periodic_length_must_be_a_multiple_of_the_cell_size(sph):
    """include/sph.h: a periodic length must be an integer multiple of the cell size (A15); otherwise particles
    would interact across a gap.  L = 1.0 with cs = 2h = 0.0832 is not; with cell_size = L / 12 it is."""
    h = C.c_void_p()
    p = _params(sph)
    p.periodic[:] = [1, 0, 0]
    assert sph.lib.sph_create(C.byref(p), C.byref(h)) == sph.SPH_E_BADARG and not h.value
    assert b"periodic length" in sph.lib.sph_last_error(None)
    p.cell_size = 1.0 / 12.0
    rc = sph.lib.sph_create(C.byref(p), C.byref(h))
    assert rc in (sph.SPH_OK, sph.SPH_E_CUDA)      # accepted (SPH_E_CUDA on a box without a GPU)
    if rc == sph.SPH_OK:
        sph.lib.sph_destroy(h)


def test_create_failure_reason_is_reported(sph):
    h = C.c_void_p()
    assert sph.lib.sph_create(C.byref(_params(sph, dim=4)), C.byref(h)) == sph.SPH_E_BADARG
    assert sph.lib.sph_last_error(None) == b"dim must be 2 or 3"


def test_null_arguments(sph):
    h = C.c_void_p()
    assert sph.lib.sph_create(None, C.byref(h)) == sph.SPH_E_BADARG
    assert sph.lib.sph_step(None, 1) == sph.SPH_E_BADARG
    assert sph.lib.sph_compute_interactions(None) == sph.SPH_E_BADARG
    sph.lib.sph_destroy(None)  # allowed


def test_grid_overflow_is_reported(sph):
    p = _params(sph)
    p.domain_max[:] = [1e4, 1e4, 1e4]   # ~1.7e15 cells
    h = C.c_void_p()
    assert sph.lib.sph_create(C.byref(p), C.byref(h)) == sph.SPH_E_OVERFLOW


def test_no_cpu_fallback(sph):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present: covered by the gpu tests")
    h = C.c_void_p()
    assert sph.lib.sph_create(C.byref(_params(sph)), C.byref(h)) == sph.SPH_E_CUDA
    with pytest.raises(sph.SphError):
        sph.Sph(dict(dim=3))


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2104_00537_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", txt, flags=re.M), f
                assert "sph_oracle" not in txt and "liborc" not in txt, f
    orc = open(os.path.join(ROOT, "oracle", "__init__.py")).read() + open(os.path.join(ROOT, "oracle", "sph_oracle.c")).read()
    assert "paper_2104_00537_b200" not in orc.replace("paper_2104_00537_b200/csrc", "")
