"""GPU parity for the option branches and host-state rules that test_gpu_parity.py does not reach:
ddt_over_boundary (A4), rho_bound_floor (A10), gamma != 7 (Eq. 28), the fall-back chains of the interaction
kernels (eta2_coef = 0, Fourtakas term outside its series range), the viscous dt candidate over accepted pairs
only (A12), reload rules, two contexts on two streams, and the device fault flag of an interaction pass.
Tolerances are those of test_gpu_parity.py (BASELINE.json north_star)."""
import numpy as np
import pytest

import oracle
from paper_2104_00537_b200 import workloads as wl
from test_gpu_parity import KERNELS, assert_close, check_one_pass, developed_state, small_params

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def sph():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_2104_00537_b200 import sph as mod
    return mod


# ---- A4: density diffusion over boundary neighbours too --------------------------------------------------
@pytest.mark.parametrize("pi_kernel", KERNELS)
@pytest.mark.parametrize("ddt_model", [0, 1])
def test_ddt_over_boundary(sph, pi_kernel, ddt_model):
    c = developed_state(wl.config(0), 4)
    c.params.update(ddt_over_boundary=1, ddt_model=ddt_model)
    ref = oracle.State(c.params, c.pos, c.vel, c.rho, c.ptype).interactions()
    ref0 = oracle.State(dict(c.params, ddt_over_boundary=0), c.pos, c.vel, c.rho, c.ptype).interactions()
    fl = c.ptype == 0
    assert np.abs(ref["drho"][fl] - ref0["drho"][fl]).max() > 1e-3 * np.abs(ref["drho"][fl]).max()   # it matters
    check_one_pass(sph, c, pi_kernel)


# ---- A10: boundary density floored at rho0 ---------------------------------------------------------------
@pytest.mark.parametrize("integrator", [0, 1])
def test_rho_bound_floor_steps(sph, integrator):
    c = wl.config(0)
    c.params.update(rho_bound_floor=1)
    st = oracle.State(c.params, c.pos, c.vel, c.rho, c.ptype)
    st0 = oracle.State(dict(c.params, rho_bound_floor=0), c.pos, c.vel, c.rho, c.ptype)
    if integrator == 0:
        st.step(10); st0.step(10)
    else:
        st.step_verlet(10, 4); st0.step_verlet(10, 4)
    bd = c.ptype != 0
    assert (st0.rho[bd] < c.params["rho0"]).any() and (st.rho[bd] >= c.params["rho0"]).all()   # the clamp acts here
    with sph.Sph(dict(c.params, integrator=integrator, verlet_steps=4)) as S:
        S.load_case(c)
        S.step(10)
        assert np.abs(S.read_state(sph.SPH_POS) - st.pos).max() <= 1e-3 * c.params["dp"]
        rho = S.read_state(sph.SPH_RHO).astype(np.float64)
        assert (rho[bd] >= c.params["rho0"]).all()
        assert_close("rho", rho, st.rho, rtol=1e-5, floor=0)
        assert abs(rho.sum() - st.rho.sum()) <= 1e-6 * st.rho.sum()


# ---- Eq. 28 with gamma != 7 (the expm1/log1p branch of the library's EOS) ---------------------------------
@pytest.mark.parametrize("pi_kernel", KERNELS)
def test_gamma_5(sph, pi_kernel):
    c = developed_state(wl.config(0), 4)
    c.params.update(gamma=5.0)
    check_one_pass(sph, c, pi_kernel)      # compares SPH_PRESS with oracle.eos at rel 2e-6, and every sum


def test_gamma_5_steps(sph):
    c = wl.config(0)
    c.params.update(gamma=5.0)
    st = oracle.State(c.params, c.pos, c.vel, c.rho, c.ptype).step(8)
    with sph.Sph(c.params) as S:
        S.load_case(c)
        S.step(8)
        assert np.abs(S.read_state(sph.SPH_POS) - st.pos).max() <= 1e-3 * c.params["dp"]
        assert_close("rho", S.read_state(sph.SPH_RHO), st.rho, rtol=1e-5, floor=0)


# ---- fall-back chains of the interaction kernels -----------------------------------------------------------
def test_eta2_zero_falls_through_to_gather(sph):
    """eta^2 = 0: the quad and tiled kernels rely on eta^2 > 0 for the self pair and refuse; auto must end at the
    gather kernel with the same results."""
    c = developed_state(wl.config(0), 3)
    c.params.update(eta2_coef=0.0)
    for pk in (0, 3, 2, 1):
        info = check_one_pass(sph, c, pk)
        assert info.pi_kernel == 1


def test_fourtakas_outside_series_range(sph):
    """ddt_model = 1 with rho0 |g| 2h / B > 0.02: the packed series form of the inverse EOS is not exact to fp32
    there, the quad kernel refuses, and the tiled and gather kernels evaluate expm1(log1p(e) / gamma) (A23)."""
    c = developed_state(wl.config(0), 3)
    c.params.update(ddt_model=1, g=(0.0, 0.0, -40.0))
    p = c.params
    assert p["rho0"] * 40.0 * 2 * p["h"] / (p["c0"] ** 2 * p["rho0"] / p["gamma"]) > 0.02
    for pk, ran in ((0, 2), (3, 2), (2, 2), (1, 1)):
        info = check_one_pass(sph, c, pk)
        assert info.pi_kernel == ran


# ---- A12: the viscous dt candidate runs over accepted pairs only --------------------------------------------
def test_dt_ignores_pairs_outside_the_support(sph):
    """A block in uniform translation (every accepted pair has v_ab = 0, so max |mu_ab| = 0) next to a sheet of
    fast particles just outside everyone's support: candidates of the cell search, but not neighbours.  dt must be
    CFL min(sqrt(h/|g|), h/c0) whichever kernel runs, and identical across the three kernels."""
    p = small_params()
    dp, h = p["dp"], p["h"]
    n1 = 10
    ii = np.stack(np.meshgrid(np.arange(n1), np.arange(n1), np.arange(n1), indexing="ij"), -1).reshape(-1, 3)
    block = 0.1 + (ii + 0.5) * dp
    x_sheet = block[:, 0].max() + 2.0 * h * 1.02
    jj = np.stack(np.meshgrid(np.arange(4), np.arange(4), indexing="ij"), -1).reshape(-1, 2)
    sheet = np.stack([np.full(len(jj), x_sheet), 0.12 + jj[:, 0] * 2.5 * h, 0.12 + jj[:, 1] * 2.5 * h], 1)
    pos = np.concatenate([block, sheet])
    vel = np.zeros_like(pos, dtype=np.float32)
    vel[:len(block)] = (1.0, 0.5, 0.0)
    vel[len(block):] = (-40.0, 0.0, 25.0)
    rho = np.full(len(pos), 1000.0, np.float32)
    typ = np.zeros(len(pos), np.uint8)
    c = wl.Case("translation", pos, vel, rho, typ, p)
    st = oracle.State(p, pos, vel, rho, typ)
    ref = st.interactions()
    assert ref["nbcount"][len(block):].sum() == 0 and ref["viscmax"] == 0.0
    dt_ref = oracle.dt(p, ref["acc"], st.ptype, st.out, ref["viscmax"])
    dts = []
    for pk in KERNELS:
        with sph.Sph(p, pi_kernel=pk, count_neighbours=True) as S:
            S.load_case(c)
            S.compute_interactions()
            info = S.get_info()
            assert info.pi_kernel == pk
            assert np.array_equal(S.read_state(sph.SPH_NBCOUNT), ref["nbcount"])
            dts.append(info.dt)
    assert dts[0] == dts[1] == dts[2]
    assert dts[0] == pytest.approx(dt_ref, rel=1e-6)


# ---- host-state rules ----------------------------------------------------------------------------------------
def test_reload_resets_the_pass_guards(sph):
    c = wl.config(0)
    with sph.Sph(c.params, count_neighbours=True) as S:
        S.load_case(c)
        S.compute_interactions()
        S.read_state(sph.SPH_ACC)
        S.load_case(c)                                   # second load, same size: no reallocation
        for f in (sph.SPH_ACC, sph.SPH_DRHODT, sph.SPH_NBCOUNT, sph.SPH_KEY, sph.SPH_CELLSTART):
            with pytest.raises(sph.SphError) as e:
                S.read_state(f)
            assert e.value.code == sph.SPH_E_STATE
        S.load_particles(np.zeros((0, 3)), np.zeros((0, 3), np.float32), np.zeros(0, np.float32), np.zeros(0, np.uint8))
        big = wl.config(2, scale=0.2)                    # larger: reallocation path
        S.load_case(big)
        S.compute_interactions()
        assert S.read_state(sph.SPH_ACC).shape == (big.n, 3)


def test_two_contexts_on_two_streams(sph):
    """Two contexts in one process, each on its own stream, stepped alternately: same results as alone."""
    import torch
    c = wl.config(0)
    st = oracle.State(c.params, c.pos, c.vel, c.rho, c.ptype).step(4)
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    with sph.Sph(c.params, stream=s1) as A, sph.Sph(c.params, pi_kernel=2, stream=s2) as B:
        A.load_case(c); B.load_case(c)
        for _ in range(4):
            A.step(1); B.step(1)
        for S, pk in ((A, 3), (B, 2)):
            assert S.get_info().pi_kernel == pk
            assert np.abs(S.read_state(sph.SPH_POS) - st.pos).max() <= 1e-3 * c.params["dp"]
            assert_close("rho", S.read_state(sph.SPH_RHO), st.rho, rtol=1e-5, floor=0)


@pytest.mark.parametrize("pi_kernel", KERNELS)
def test_nan_is_flagged_by_an_interaction_pass(sph, pi_kernel):
    p = small_params()
    with sph.Sph(p, pi_kernel=pi_kernel) as S:
        n = 200
        rho = np.full(n, 1000.0, np.float32)
        rho[7] = np.nan
        pos = 0.2 + 0.08 * np.stack([wl.uniform01(1, np.arange(n), k) for k in range(3)], 1)
        S.load_particles(pos, np.zeros((n, 3), np.float32), rho, np.zeros(n, np.uint8))
        S.compute_interactions()
        with pytest.raises(sph.SphError) as e:
            S.get_info()
        assert e.value.code == sph.SPH_E_NAN


# ---- sph_read_fields: several fields, one synchronisation; same bytes as field-by-field reads ---------------
def test_read_fields_matches_single_reads_and_checks_before_launch(sph):
    import ctypes as C
    c = developed_state(wl.config(0), 2)
    with sph.Sph(c.params, count_neighbours=True) as S:
        S.load_case(c)
        S.step(2)
        S.compute_interactions()
        n = S.n
        want = {f: S.read_state(f) for f in (sph.SPH_POS, sph.SPH_VEL, sph.SPH_RHO, sph.SPH_ACC, sph.SPH_NBCOUNT,
                                             sph.SPH_KEY, sph.SPH_PERM)}
        got = {f: np.empty_like(a) for f, a in want.items()}
        fields = list(want)
        S.read_fields_ptr(fields, [got[f].ctypes.data for f in fields], [got[f].nbytes for f in fields])
        for f in fields:
            assert np.array_equal(got[f], want[f]), f
        # one short buffer fails the whole call before anything is written
        sentinel = np.full((n, 3), 7.0)
        small = np.empty(3, np.float32)
        with pytest.raises(sph.SphError) as ei:
            S.read_fields_ptr([sph.SPH_POS, sph.SPH_RHO], [sentinel.ctypes.data, small.ctypes.data],
                              [sentinel.nbytes, small.nbytes])
        assert ei.value.code == sph.SPH_E_OVERFLOW and (sentinel == 7.0).all()
        S.read_fields_ptr([], [], [])          # no-op
        # a reload after a larger case reuses the staging buffer; results are those of a fresh context
        S.load_case(c)
        S.step(1)
        again = S.read_state(sph.SPH_POS)
    with sph.Sph(c.params) as T:
        T.load_case(c)
        T.step(1)
        assert np.array_equal(again, T.read_state(sph.SPH_POS))
