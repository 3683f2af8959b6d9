"""Parity of the NEXT-3 (mDBC, Eq. 38-39) and NEXT-4 (particle shifting, Eq. 40-41, 53-54) CUDA passes against the
CPU oracle, through the C ABI, on the same seeded inputs.

Tolerances: the standard ones of test_gpu_parity.py (rel 1e-4 with floor 1e-6 * max|value| per particle after one
call; positions <= 1e-3 dp after ten steps).  The mDBC density is compared as rho_B - rho0 (the quantity the pressure
depends on) at rel 1e-4 with floor 1e-6 * rho0: rho itself is an fp32 state variable with spacing 6e-8 * rho0.
"""
import numpy as np
import pytest

import oracle
from paper_2104_00537_b200 import workloads as wl

pytestmark = pytest.mark.gpu

KERNELS = [1, 2, 3]


@pytest.fixture(scope="module")
def sph():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_2104_00537_b200 import sph as mod
    return mod


def assert_close(name, got, ref, rtol=1e-4, floor=1e-6, scale=None):
    got = np.asarray(got, np.float64)
    ref = np.asarray(ref, np.float64)
    if scale is None:
        scale = np.abs(ref).max() if ref.size else 0.0
    err = np.abs(got - ref)
    tol = rtol * np.abs(ref) + floor * scale
    bad = err > tol
    assert not bad.any(), (f"{name}: {bad.sum()} of {bad.size} outside rel {rtol} / floor {floor}*{scale:.3e}; "
                           f"worst err {err.max():.3e} (ref {ref.ravel()[err.argmax()]:.6e})")


def perturbed(case, seed, rho_sigma=3.0, vel_sigma=0.1):
    """The case with a seeded, fp32-rounded density and velocity field (a state with gradients everywhere)."""
    idx = np.arange(case.n)
    z = case.pos[:, 2]
    rho = (1000.0 + 25.0 * (z.max() - z) + rho_sigma * wl.normal01(seed, idx, 1)).astype(np.float32)
    vel = (vel_sigma * np.stack([wl.normal01(seed, idx, 2 + k) for k in range(3)], axis=1)).astype(np.float32)
    if case.params["dim"] == 2:
        vel[:, 1] = 0.0
    vel[case.ptype != 0] = 0.0
    return wl.Case(case.name + "_pert", case.pos, vel, rho, case.ptype, dict(case.params), motions=list(case.motions),
                   normals=case.normals, box=case.box)


def with_piston(case):
    """The wall x < 0 of a tank becomes moving group 2 (imposed motion along x)."""
    typ = case.ptype.copy()
    typ[(typ != 0) & (case.pos[:, 0] < 0)] = 2
    c = wl.Case(case.name + "_piston", case.pos, case.vel, case.rho, typ, dict(case.params),
                motions=[dict(group=2, axis=0, stroke=0.05, period=0.08, phase=0.4)], normals=case.normals, box=case.box)
    return c


# ---- mDBC -----------------------------------------------------------------------------------------------------------
def check_mdbc_one_pass(sph, case, pi_kernel, slip):
    p = dict(case.params, boundary_model=1, mdbc_slip=slip)
    st = oracle.State(p, case.pos, case.vel, case.rho, case.ptype, motions=case.motions, normals=case.normals)
    vwall = np.zeros((case.n, 3))
    for m in case.motions:      # the wall velocity at t = 0, from the closed form of Eq. 37 (pinned on the oracle side)
        vwall[case.ptype == m["group"], m["axis"]] = 0.5 * m["stroke"] * 2 * np.pi / m["period"] * np.cos(m["phase"])
    vel_m, rho_m, status = oracle.mdbc(p, st.cell, st.u, st.out, st.vel, st.rho, st.ptype, case.normals, vwall=vwall)
    ref = oracle.interactions(p, st.cell, st.u, st.out, vel_m, rho_m, st.ptype, mode=1)
    bnd = (case.ptype != 0) & (st.out == 0)
    with sph.Sph(p, pi_kernel=pi_kernel, count_neighbours=True) as S:
        S.load_case(case)
        S.compute_interactions()
        rho = S.read_state(sph.SPH_RHO).astype(np.float64)
        assert_close("rho_B - rho0", rho[bnd] - 1000.0, rho_m[bnd] - 1000.0, scale=1000.0)
        np.testing.assert_array_equal(rho[~bnd], case.rho[~bnd])              # fluid untouched
        assert_close("v_B", S.read_state(sph.SPH_VEL)[bnd], vel_m[bnd], floor=1e-5)
        P_ref = np.array([oracle.eos(p, float(np.float32(r))) for r in rho_m[bnd][:3000]])
        assert_close("P_B", S.read_state(sph.SPH_PRESS)[bnd][:3000], P_ref, rtol=2e-4, floor=1e-5)
        act = st.out == 0
        assert np.array_equal(S.read_state(sph.SPH_NBCOUNT)[act], ref["nbcount"][act])
        assert_close("acc", S.read_state(sph.SPH_ACC)[act], ref["acc"][act])
        assert_close("drho", S.read_state(sph.SPH_DRHODT)[act], ref["drho"][act])
        # idempotent: a second call on the same state gives the same boundary state
        S.compute_interactions()
        np.testing.assert_array_equal(S.read_state(sph.SPH_RHO).astype(np.float64), rho)
    return status


@pytest.mark.parametrize("pi_kernel", KERNELS)
@pytest.mark.parametrize("slip", [0, 1])
def test_mdbc_config0_perturbed(sph, pi_kernel, slip):
    status = check_mdbc_one_pass(sph, perturbed(wl.config(0), 31), pi_kernel, slip)
    vals = set(np.unique(status))
    assert {1, 3} <= vals            # full solves next to the block, rho0 far from any fluid


@pytest.mark.parametrize("cell_div", [1, 2])
def test_mdbc_2d_and_cell_div(sph, cell_div):
    c = wl.dam_break("db2", 2, 0.02, (120, 1, 60), (40, 1, 40), 0.2, 7, 0.8, cell_div=cell_div)
    check_mdbc_one_pass(sph, perturbed(c, 33), 0, 1)
    c = wl.config(0, cell_div=cell_div)
    check_mdbc_one_pass(sph, perturbed(c, 34), 1, 1)


@pytest.mark.parametrize("slip", [0, 1])
def test_mdbc_dam_break_with_obstacle(sph, slip):
    """The obstacle's particles carry interface vectors of their own (workloads.obstacle_normals), so their ghost nodes
    lie in the fluid around the obstacle: full solves must occur on the obstacle, not only on the tank."""
    c = wl.dam_break("obstacle", 3, 0.02, (40, 20, 20), (15, 20, 15), 0.01, 4321, 0.3, obstacle=((13, 6, 0), (5, 8, 6)))
    status = check_mdbc_one_pass(sph, perturbed(c, 37), 0, slip)
    obs = (c.ptype != 0) & (c.pos[:, 0] > 0.26) & (c.pos[:, 0] < 0.36) & (c.pos[:, 1] > 0.12) & (c.pos[:, 1] < 0.28) & \
          (c.pos[:, 2] > 0.0) & (c.pos[:, 2] < 0.12)
    assert obs.sum() == 5 * 8 * 6 and (status[obs] == 1).sum() > 20


def test_mdbc_moving_wall_no_slip(sph):
    c = with_piston(perturbed(wl.config(0), 35))
    check_mdbc_one_pass(sph, c, 3, 1)


def test_mdbc_det_threshold_and_missing_normals(sph):
    """mdbc_det_min above every determinant -> Shepard values everywhere; no normals -> ghost node on the particle."""
    c = perturbed(wl.config(0), 36)
    for extra, normals in ((dict(mdbc_det_min=50.0), c.normals), ({}, None)):
        p = dict(c.params, boundary_model=1, **extra)
        st = oracle.State(p, c.pos, c.vel, c.rho, c.ptype)
        nrm = normals if normals is not None else np.zeros_like(c.pos)
        _, rho_m, status = oracle.mdbc(p, st.cell, st.u, st.out, st.vel, st.rho, st.ptype, nrm)
        if extra:
            assert 1 not in set(np.unique(status)) and 2 in set(np.unique(status))
        with sph.Sph(p, pi_kernel=1) as S:
            S.load_particles(c.pos, c.vel, c.rho, c.ptype)
            if normals is not None:
                S.set_boundary_normals(normals)
            S.compute_interactions()
            bnd = c.ptype != 0
            assert_close("rho_B - rho0", S.read_state(sph.SPH_RHO).astype(np.float64)[bnd] - 1000.0, rho_m[bnd] - 1000.0,
                         scale=1000.0)


@pytest.mark.parametrize("pi_kernel", KERNELS)
@pytest.mark.parametrize("integrator", [0, 1])
def test_mdbc_ten_steps(sph, pi_kernel, integrator):
    c = with_piston(wl.config(0))
    p = dict(c.params, boundary_model=1, mdbc_slip=1, integrator=integrator, verlet_steps=4)
    st = oracle.State(p, c.pos, c.vel, c.rho, c.ptype, motions=c.motions, normals=c.normals)
    st.step(10) if integrator == 0 else st.step_verlet(10, 4)
    with sph.Sph(p, pi_kernel=pi_kernel) as S:
        S.load_case(c)
        S.step(10)
        info = S.get_info()
        assert info.steps_done == 10 and info.n_out == 0
        assert info.t == pytest.approx(st.t, rel=1e-5)
        assert np.abs(S.read_state(sph.SPH_POS) - st.pos).max() <= 1e-3 * p["dp"]
        rho = S.read_state(sph.SPH_RHO).astype(np.float64)
        assert abs(rho.sum() - st.rho.sum()) <= 1e-6 * st.rho.sum()
        assert_close("rho - rho0", rho - 1000.0, st.rho - 1000.0, rtol=1e-3, floor=1e-5, scale=1000.0)
        assert_close("vel", S.read_state(sph.SPH_VEL), st.vel, rtol=1e-4, floor=1e-4)
        tm = S.get_timings()
        assert tm.n_interaction_passes == (20 if integrator == 0 else 10)


def test_mdbc_hydrostatic_column_keeps_the_wall_pressure_continuous(sph):
    """Physics band (not a parity pin): on a resting hydrostatic column the mDBC wall particles under the floor take the
    hydrostatic density continued into the wall (rho_B rises with depth below the interface), as Eq. 38 intends."""
    c = wl.hydrostatic_column("col", 0.02, (12, 12, 30), 20)
    p = dict(c.params, boundary_model=1)
    with sph.Sph(p) as S:
        S.load_case(c)
        S.compute_interactions()
        rho = S.read_state(sph.SPH_RHO).astype(np.float64)
    floor1 = (c.ptype != 0) & (np.abs(c.pos[:, 2] + 0.5 * 0.02) < 1e-9) & (np.abs(c.pos[:, 0] - 0.13) < 0.05) & \
             (np.abs(c.pos[:, 1] - 0.13) < 0.05)
    floor2 = (c.ptype != 0) & (np.abs(c.pos[:, 2] + 1.5 * 0.02) < 1e-9) & (np.abs(c.pos[:, 0] - 0.13) < 0.05) & \
             (np.abs(c.pos[:, 1] - 0.13) < 0.05)
    bottom = (c.ptype == 0) & (np.abs(c.pos[:, 2] - 0.5 * 0.02) < 1e-9)
    assert floor1.sum() > 0 and floor2.sum() > 0
    assert rho[floor2].mean() > rho[floor1].mean() > rho[bottom].mean()


# ---- particle shifting ------------------------------------------------------------------------------------------------
def check_shift_one_pass(sph, case, pi_kernel, **extra):
    p = dict(case.params, shift_model=1, shift_coef=2.0, **extra)
    st = oracle.State(p, case.pos, case.vel, case.rho, case.ptype)
    conc = oracle.concentration(p, st.cell, st.u, st.out, st.rho, st.ptype)
    shift, gradc = oracle.shift_velocity(p, st.cell, st.u, st.out, st.vel, st.rho, st.ptype, conc)
    ref = st.interactions()
    act = st.out == 0
    with sph.Sph(p, pi_kernel=pi_kernel) as S:
        S.load_case(case)
        with pytest.raises(sph.SphError) as e:
            S.read_state(sph.SPH_SHIFT)
        assert e.value.code == sph.SPH_E_STATE
        S.compute_interactions()
        assert_close("C", S.read_state(sph.SPH_CONC)[act], conc[act], rtol=1e-6, floor=0)
        assert_close("shift", S.read_state(sph.SPH_SHIFT)[act], shift[act])
        assert_close("acc", S.read_state(sph.SPH_ACC)[act], ref["acc"][act])          # the main pass is unchanged
    return conc, shift


@pytest.mark.parametrize("pi_kernel", KERNELS)
def test_shift_config0_perturbed(sph, pi_kernel):
    conc, shift = check_shift_one_pass(sph, perturbed(wl.config(0), 41, vel_sigma=0.3), pi_kernel)
    assert conc.min() < 0.7 and conc.max() > 0.99 and np.abs(shift).max() > 0


@pytest.mark.parametrize("extra", [dict(shift_fs_conc=0.9), dict(shift_fs_conc=0.9, shift_alpha_n=0.1, shift_beta_n=2.0)])
def test_shift_free_surface_form(sph, extra):
    c = perturbed(wl.config(0), 42, vel_sigma=0.3)
    conc, shift = check_shift_one_pass(sph, c, 0, **extra)
    fs = (conc < 0.9) & (c.ptype == 0)
    assert fs.sum() > 100
    if "shift_alpha_n" not in extra:
        assert np.all(shift[fs] == 0.0)


@pytest.mark.parametrize("dim,periodic,cell_div", [(2, (0, 0, 0), 1), (3, (1, 1, 1), 1), (3, (0, 0, 0), 2), (2, (1, 0, 1), 2)])
def test_shift_random_clouds(sph, dim, periodic, cell_div):
    box = (0.9, 0.9, 0.9) if dim == 3 else (2.4, 0.0, 2.4)
    c = wl.random_cloud("rc", 9973 if dim == 3 else 6007, box, 0.02, 77 + dim + cell_div, dim=dim, periodic=periodic,
                        cell_div=cell_div)
    check_shift_one_pass(sph, c, 0)


def test_shift_fields_are_zero_for_particles_out_of_the_grid(sph):
    """include/sph.h: SPH_CONC and SPH_SHIFT are 0 for particles out of the grid (A16), as in the oracle, which skips
    them.  The first pass fills every sorted slot; after the reload three fluid particles have left the grid, and their
    slots (sorted last, C3) must not keep what other particles left there."""
    c = perturbed(wl.config(0), 45, vel_sigma=0.3)
    p = dict(c.params, shift_model=1, shift_coef=2.0)
    esc = np.flatnonzero(c.ptype == 0)[[5, 600, 4000]]
    pos2 = c.pos.copy()
    pos2[esc, 2] += 50.0
    st = oracle.State(p, pos2, c.vel, c.rho, c.ptype)
    assert st.out.sum() == 3 and (st.out[esc] == 1).all()
    conc = oracle.concentration(p, st.cell, st.u, st.out, st.rho, st.ptype)
    shift, _ = oracle.shift_velocity(p, st.cell, st.u, st.out, st.vel, st.rho, st.ptype, conc)
    assert (conc[esc] == 0).all() and (shift[esc] == 0).all()
    with sph.Sph(p) as S:
        S.load_case(c)
        S.compute_interactions()
        assert (S.read_state(sph.SPH_CONC) > 0).all()
        S.load_particles(pos2, c.vel, c.rho, c.ptype)
        S.compute_interactions()
        assert S.get_info().n_out == 3
        got_c, got_s = S.read_state(sph.SPH_CONC), S.read_state(sph.SPH_SHIFT)
        assert (got_c[esc] == 0).all() and (got_s[esc] == 0).all()
        assert_close("C", got_c, conc, rtol=1e-6, floor=0)          # every particle, the escaped ones included
        assert_close("shift", got_s, shift)


@pytest.mark.parametrize("pi_kernel", KERNELS)
@pytest.mark.parametrize("integrator", [0, 1])
def test_shift_ten_steps(sph, pi_kernel, integrator):
    c = perturbed(wl.config(0), 43, rho_sigma=0.0, vel_sigma=0.2)
    c.rho[:] = 1000.0
    p = dict(c.params, shift_model=1, shift_coef=2.0, shift_fs_conc=0.85, integrator=integrator, verlet_steps=4)
    st = oracle.State(p, c.pos, c.vel, c.rho, c.ptype)
    st.step(10) if integrator == 0 else st.step_verlet(10, 4)
    off = oracle.State(dict(p, shift_model=0), c.pos, c.vel, c.rho, c.ptype)
    off.step(10) if integrator == 0 else off.step_verlet(10, 4)
    with sph.Sph(p, pi_kernel=pi_kernel) as S:
        S.load_case(c)
        S.step(10)
        pos = S.read_state(sph.SPH_POS)
        assert np.abs(pos - st.pos).max() <= 1e-3 * p["dp"]
        assert np.abs(pos - off.pos).max() > 1e-2 * p["dp"]           # the shift is far above the tolerance
        assert_close("vel", S.read_state(sph.SPH_VEL), st.vel, rtol=1e-4, floor=1e-4)
        tm = S.get_timings()
        assert tm.ms_shift == 0.0 and tm.n_interaction_passes == (20 if integrator == 0 else 10)


def test_mdbc_with_shifting_and_options_together(sph):
    """Everything on: mDBC no-slip with a piston, shifting with the free-surface form, laminar viscosity, Fourtakas DDT."""
    c = with_piston(wl.config(0))
    p = dict(c.params, boundary_model=1, mdbc_slip=1, shift_model=1, shift_coef=3.0, shift_fs_conc=0.85,
             visco_model=1, nu0=1e-3, ddt_model=1)
    st = oracle.State(p, c.pos, c.vel, c.rho, c.ptype, motions=c.motions, normals=c.normals).step(6)
    with sph.Sph(p) as S:
        S.load_case(c)
        S.step(6)
        assert np.abs(S.read_state(sph.SPH_POS) - st.pos).max() <= 1e-3 * p["dp"]
        assert_close("vel", S.read_state(sph.SPH_VEL), st.vel, rtol=1e-4, floor=1e-4)


def test_normals_call_order(sph):
    c = wl.config(0)
    with sph.Sph(dict(c.params, boundary_model=1)) as S:
        with pytest.raises(sph.SphError) as e:
            S.n = c.n
            S.set_boundary_normals(c.normals)
        assert e.value.code == sph.SPH_E_STATE
