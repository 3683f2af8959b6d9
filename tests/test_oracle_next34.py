"""Pins for the NEXT-3 (mDBC, Eq. 38-39) and NEXT-4 (particle shifting, Eq. 40-41 at
PAPER.md:326-334 with Eq. 53-54 at 434-442) parts of the CPU oracle, against what the mathematics fixes.
None of these call the CUDA library.
"""
import math

import numpy as np
import pytest

import oracle
from paper_2104_00537_b200 import workloads as wl

DP = 0.02
H3 = 1.2 * math.sqrt(3) * DP
H2 = 1.2 * math.sqrt(2) * DP


def params(dim=3, **kw):
    p = wl._params(dim, DP, 1.2, 10 * math.sqrt(9.81 * 0.3), (0, 0, 0), (-0.4, -0.4 if dim == 3 else 0.0, -0.4),
                   (0.4, 0.4 if dim == 3 else 0.0, 0.4))
    p.update(kw)
    return p


def half_space_cloud(dim, seed=5, jitter=0.3, nside=12):
    """Jittered fluid lattice filling z > 0 around the origin (no symmetry left), plus one wall particle below."""
    r = (np.arange(nside) - nside / 2 + 0.5) * DP
    z = (np.arange(nside // 2) + 0.5) * DP
    if dim == 3:
        X, Y, Z = np.meshgrid(r, r, z, indexing="ij")
        pos = np.stack([X.ravel(), Y.ravel(), Z.ravel()], axis=1)
    else:
        X, Z = np.meshgrid(r, z, indexing="ij")
        pos = np.stack([X.ravel(), 0 * X.ravel(), Z.ravel()], axis=1)
    idx = np.arange(len(pos))
    for ax in range(3):
        if dim == 2 and ax == 1:
            continue
        pos[:, ax] += (2 * wl.uniform01(seed, idx, ax) - 1) * jitter * DP
    pos[:, 2] = np.abs(pos[:, 2]) + 1e-3 * DP
    return pos


# ---- mDBC ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dim", [3, 2])
def test_mdbc_reproduces_a_linear_density_field_exactly(dim):
    """The corrected approximation of Liu & Liu is exact for linear fields on ANY particle arrangement: with
    rho_b = c + k . r_b the ghost node gets rho_G = c + k . r_G and Eq. 38 returns rho_B = c + k . r_B, the linear
    field continued to the boundary particle.  A constant field (k = 0) comes back with zero gradient."""
    fpos = half_space_cloud(dim)
    bpos = np.array([[0.003, 0.001 if dim == 3 else 0.0, -0.5 * DP], [0.1, 0.0, -1.5 * DP]])
    nrm = np.array([[0.0, 0.0, 0.5 * DP], [0.0, 0.0, 1.5 * DP]])
    pos = np.concatenate([bpos, fpos])
    typ = np.concatenate([np.ones(2, np.uint8), np.zeros(len(fpos), np.uint8)])
    normals = np.concatenate([nrm, np.zeros_like(fpos)])
    p = params(dim)
    cell, u, out = oracle.canonicalize(p, pos)
    x = oracle.position(p, cell, u)                      # the oracle's true positions
    for c, k in ((1000.0, np.array([35.0, -20.0 if dim == 3 else 0.0, 60.0])), (1003.0, np.zeros(3))):
        rho = c + x @ k
        rho[:2] = 777.0                                  # whatever the boundary particles held is ignored
        for mode in (0, 1):
            _, rho_out, status = oracle.mdbc(p, cell, u, out, np.zeros_like(pos), rho, typ, normals, mode=mode)
            assert list(status[:2]) == [1, 1]
            np.testing.assert_allclose(rho_out[:2], c + x[:2] @ k, rtol=1e-10)
            np.testing.assert_array_equal(rho_out[2:], rho[2:])          # fluid untouched


def test_mdbc_matrix_against_numpy_solve():
    """One ghost node, the (d+1) x (d+1) system assembled and solved independently with numpy on a NON-linear field
    (rho = rho0 + 40 sin(12 z) + 900 x y): pins the assembly, the solve and the Eq. 38 extrapolation."""
    fpos = half_space_cloud(3, seed=9)
    bpos = np.array([[0.004, -0.002, -0.5 * DP]])
    nrm = np.array([[0.0, 0.0, 0.5 * DP]])
    pos = np.concatenate([bpos, fpos])
    typ = np.concatenate([np.ones(1, np.uint8), np.zeros(len(fpos), np.uint8)])
    p = params(3)
    cell, u, out = oracle.canonicalize(p, pos)
    x = oracle.position(p, cell, u)
    rho = 1000.0 + 40 * np.sin(12 * x[:, 2]) + 900 * x[:, 0] * x[:, 1]
    _, rho_out, status = oracle.mdbc(p, cell, u, out, np.zeros_like(pos), rho, typ,
                                     np.concatenate([nrm, np.zeros_like(fpos)]), mode=1)
    m = 1000.0 * DP ** 3
    xg = x[0] + 2 * nrm[0]
    d = x[1:] - xg
    r = np.linalg.norm(d, axis=1)
    sel = r < 2 * H3
    d, r, rb = d[sel], r[sel], rho[1:][sel]
    W = np.array([oracle.W(3, H3, float(t)) for t in r])
    f = np.array([oracle.fab(3, H3, float(t)) for t in r])
    gW = -f[:, None] * d
    V = m / rb
    basis = np.concatenate([np.ones((len(d), 1)), d], axis=1)          # (1, d)
    test = np.concatenate([W[:, None], gW], axis=1)                    # (W, grad W)
    A = (test * V[:, None]).T @ basis
    b = (test * V[:, None]).T @ rb
    sol = np.linalg.solve(A, b)
    assert status[0] == 1 and abs(np.linalg.det(A)) > 1e-3
    assert rho_out[0] == pytest.approx(sol[0] + (x[0] - xg) @ sol[1:], rel=1e-11)
    assert 0.05 < np.linalg.det(A) < 1.0      # a half-filled support: far above the 1e-3 threshold, below the full-support value 1


def test_mdbc_ghost_node_sits_at_twice_the_normal():
    """A lone fluid particle 0.9 * 2h above the wall particle along the normal direction, normal length 0.45 * 2h:
    only a ghost node at r_B + 2 n (0.9 * 2h up) reaches it; r_B + n or r_B would leave rho0 (status 3)."""
    p = params(3)
    R = 2 * H3
    pos = np.array([[0.0, 0.0, -0.01], [0.0, 0.0, -0.01 + 0.9 * R + 0.5 * R]])
    typ = np.array([1, 0], np.uint8)
    cell, u, out = oracle.canonicalize(p, pos)
    rho = np.array([1000.0, 1012.0])
    for nz, want_status, want_rho in ((0.45 * R, 2, 1012.0), (0.15 * R, 3, 1000.0)):
        nrm = np.array([[0.0, 0.0, nz], [0, 0, 0]])
        for mode in (0, 1):
            _, rho_out, status = oracle.mdbc(p, cell, u, out, np.zeros_like(pos), rho, typ, nrm, mode=mode)
            assert status[0] == want_status
            assert rho_out[0] == pytest.approx(want_rho, rel=1e-12)      # one neighbour: Shepard value = its density


def test_mdbc_fallbacks_shepard_and_no_neighbour():
    """Few coplanar neighbours make the system singular (det = 0 < mdbc_det_min): the Shepard value
    sum m W / sum V W, no gradient (reading A25); det threshold above every determinant -> Shepard everywhere."""
    p = params(3)
    fz = 0.6 * DP
    fpos = np.array([[0.0, 0.0, fz], [DP, 0.0, fz], [0.0, DP, fz], [-DP, -DP, fz]])     # all in the plane z = fz
    pos = np.concatenate([[[0.0, 0.0, -0.5 * DP]], fpos])
    typ = np.array([1, 0, 0, 0, 0], np.uint8)
    nrm = np.zeros_like(pos); nrm[0, 2] = 0.5 * DP
    rho = np.array([0.0, 1001.0, 1003.0, 1005.0, 1011.0])
    cell, u, out = oracle.canonicalize(p, pos)
    x = oracle.position(p, cell, u)
    _, rho_out, status = oracle.mdbc(p, cell, u, out, np.zeros_like(pos), rho, typ, nrm, mode=0)
    xg = x[0] + 2 * nrm[0]
    W = np.array([oracle.W(3, H3, float(np.linalg.norm(x[i] - xg))) for i in range(1, 5)])
    V = 1.0 / rho[1:]
    assert status[0] == 2
    assert rho_out[0] == pytest.approx(W.sum() / (V * W).sum(), rel=1e-12)
    # a well-conditioned case forced to the fallback by the threshold
    fpos = half_space_cloud(3)
    pos = np.concatenate([[[0.0, 0.0, -0.5 * DP]], fpos])
    typ = np.concatenate([np.ones(1, np.uint8), np.zeros(len(fpos), np.uint8)])
    nrm = np.zeros_like(pos); nrm[0, 2] = 0.5 * DP
    cell, u, out = oracle.canonicalize(p, pos)
    x = oracle.position(p, cell, u)
    rho = 1000.0 + 60.0 * x[:, 2]
    _, r1, s1 = oracle.mdbc(p, cell, u, out, np.zeros_like(pos), rho, typ, nrm, mode=1)
    _, r2, s2 = oracle.mdbc(dict(p, mdbc_det_min=10.0), cell, u, out, np.zeros_like(pos), rho, typ, nrm, mode=1)
    assert (s1[0], s2[0]) == (1, 2)
    assert r1[0] == pytest.approx(1000.0 + 60.0 * x[0, 2], rel=1e-10)
    xg = x[0] + 2 * nrm[0]
    d = np.linalg.norm(x[1:] - xg, axis=1)
    W = np.array([oracle.W(3, H3, float(t)) if t < 2 * H3 else 0.0 for t in d])
    assert r2[0] == pytest.approx((W.sum()) / ((W / rho[1:]).sum()), rel=1e-11)
    assert r2[0] > r1[0] + 0.5                     # the Shepard value sits at the fluid side, not at the wall


@pytest.mark.parametrize("slip", [0, 1])
def test_mdbc_velocity_shepard_and_no_slip(slip):
    """Eq. 39: the Shepard sum of a constant velocity is that velocity; no-slip gives v_B = 2 v_wall - v_G
    (= -v_G for a fixed wall), mdbc_slip = 0 leaves the imposed wall velocity."""
    fpos = half_space_cloud(3)
    pos = np.concatenate([[[0.0, 0.0, -0.5 * DP]], fpos])
    typ = np.concatenate([np.ones(1, np.uint8), np.zeros(len(fpos), np.uint8)])
    nrm = np.zeros_like(pos); nrm[0, 2] = 0.5 * DP
    p = params(3, mdbc_slip=slip)
    cell, u, out = oracle.canonicalize(p, pos)
    x = oracle.position(p, cell, u)
    v0 = np.array([0.3, -0.2, 0.05])
    vel = np.tile(v0, (len(pos), 1)); vel[0] = 9.0
    rho = 1000.0 + 5 * np.sin(40 * x[:, 0])        # non-uniform volumes
    vwall = np.zeros_like(pos); vwall[0] = [0.1, 0.0, 0.0]
    for vw in (None, vwall):
        vel_out, _, _ = oracle.mdbc(p, cell, u, out, vel, rho, typ, nrm, vwall=vw, mode=1)
        w = np.zeros(3) if vw is None else vw[0]
        want = 2 * w - v0 if slip == 1 else w
        np.testing.assert_allclose(vel_out[0], want, rtol=1e-12, atol=1e-15)
        np.testing.assert_array_equal(vel_out[1:], vel[1:])
    # a linear velocity field is NOT reproduced by the Shepard sum of a one-sided support (zeroth order only)
    vel_lin = np.stack([x[:, 2], 0 * x[:, 2], 0 * x[:, 2]], axis=1)
    if slip == 1:
        vel_out, _, _ = oracle.mdbc(p, cell, u, out, vel_lin, rho, typ, nrm, mode=1)
        xg = x[0] + 2 * nrm[0]
        d = np.linalg.norm(x[1:] - xg, axis=1)
        W = np.array([oracle.W(3, H3, float(t)) if t < 2 * H3 else 0.0 for t in d])
        V = 1.0 / rho[1:]
        assert vel_out[0, 0] == pytest.approx(-(V * W * x[1:, 2]).sum() / (V * W).sum(), rel=1e-11)


def test_mdbc_bruteforce_equals_celllist_on_a_tank_incl_periodic():
    c = wl.config(0)
    p = dict(c.params, boundary_model=1, mdbc_slip=1)
    cell, u, out = oracle.canonicalize(p, c.pos)
    idx = np.arange(c.n)
    rho = 1000.0 + 3.0 * wl.normal01(3, idx, 1)
    vel = 0.1 * np.stack([wl.normal01(3, idx, 2 + k) for k in range(3)], axis=1)
    v0, r0, s0 = oracle.mdbc(p, cell, u, out, vel, rho, c.ptype, c.normals, mode=0)
    v1, r1, s1 = oracle.mdbc(p, cell, u, out, vel, rho, c.ptype, c.normals, mode=1)
    np.testing.assert_array_equal(s0, s1)
    np.testing.assert_allclose(r0, r1, rtol=1e-12)
    np.testing.assert_allclose(v0, v1, rtol=1e-10, atol=1e-14)
    assert set(np.unique(s0[c.ptype != 0])) >= {1, 3}          # walls next to the block and walls far from any fluid
    # periodic: ghost nodes that look across the seam
    c = wl.random_cloud("rc", 3000, (0.5, 0.5, 0.5), DP, 11, periodic=(1, 1, 0))
    p = dict(c.params, boundary_model=1)
    cell, u, out = oracle.canonicalize(p, c.pos)
    nrm = 0.7 * DP * np.stack([wl.normal01(5, np.arange(c.n), k) for k in range(3)], axis=1)
    a = oracle.mdbc(p, cell, u, out, c.vel, c.rho, c.ptype, nrm, mode=0)
    b = oracle.mdbc(p, cell, u, out, c.vel, c.rho, c.ptype, nrm, mode=1)
    np.testing.assert_array_equal(a[2], b[2])
    np.testing.assert_allclose(a[1], b[1], rtol=1e-11)


@pytest.mark.parametrize("scheme", ["symplectic", "verlet"])
def test_mdbc_in_the_steppers_density_is_set_not_integrated(scheme):
    """One wall particle and one fluid particle moving away from it.  With mDBC the wall density is not integrated
    (Eq. 36 is not used); it is re-evaluated from the ghost node before every pass and keeps the value of the last
    evaluation: with one neighbour that is the Shepard value = the fluid particle's density at that pass, i.e.
    rho_f^n + dt/2 R_f^n after a symplectic step (the pass at n + 1/2) and rho_f^n after a Verlet step."""
    p = params(3, alpha=0.0, delta=0.0, boundary_model=1)
    pos = np.array([[0.0, 0.0, -0.5 * DP], [0.0, 0.0, 0.6 * DP]])
    vel = np.array([[0.0, 0, 0], [0.0, 0, 0.4]])
    typ = np.array([1, 0], np.uint8)
    nrm = np.array([[0.0, 0.0, 0.5 * DP], [0, 0, 0]])
    rho0 = np.array([990.0, 1004.0])
    st = oracle.State(p, pos, vel, rho0, typ, normals=nrm)
    first = oracle.interactions(p, st.cell, st.u, st.out, vel, np.array([1004.0, 1004.0]), typ, mode=0)
    if scheme == "symplectic":
        st.step(1)
        want = 1004.0 + 0.5 * st.dt_hist[0] * first["drho"][1]
    else:
        st.step_verlet(1, 4)
        want = 1004.0
    assert st.rho[0] == pytest.approx(want, rel=1e-13)
    assert abs(first["drho"][1]) * st.dt_hist[0] > 1e-3          # the fluid density did move
    # DBC on the same input integrates Eq. 36 instead: the wall density drops below its initial 990
    sd = oracle.State(dict(p, boundary_model=0), pos, vel, rho0, typ)
    sd.step(1) if scheme == "symplectic" else sd.step_verlet(1, 4)
    assert sd.rho[0] < 990.0 - 1e-3


# ---- particle shifting ----------------------------------------------------------------------------------------------
def lattice_case(n_side=13, dim=3):
    c = wl.periodic_cloud("lat", n_side, DP, 0.0, 5, dim=dim, vel_sigma=0.0, rho_sigma=0.0)
    c.params["g"] = (0.0, 0.0, 0.0)
    return c


def test_concentration_on_a_full_lattice_is_the_partition_of_unity():
    """C_a = sum_b V_b W_ab, self included: 1.00049 on the cubic lattice at h = 1.2 sqrt(3) dp (the same
    number test_p1_lattice_partition_of_unity obtains from orc_W alone), and grad C = 0, no shift."""
    c = lattice_case()
    p = dict(c.params, shift_model=1, shift_coef=2.0)
    cell, u, out = oracle.canonicalize(p, c.pos)
    rho = np.full(c.n, 1000.0)
    conc = oracle.concentration(p, cell, u, out, rho, c.ptype, mode=1)
    assert np.all(np.abs(conc - 1.00049) < 2e-5)
    vel = np.ones((c.n, 3))
    shift, gradc = oracle.shift_velocity(p, cell, u, out, vel, rho, c.ptype, conc, mode=1)
    # zero up to the 2^-22 position grid of C1 (relative spacing errors ~1e-7), against O(1) at a free surface
    assert np.max(np.abs(gradc)) * H3 < 1e-6 and np.max(np.abs(shift)) < 1e-5 * np.sqrt(3.0)


NS = 13      # sites per periodic axis: 3 cells of 2h (a periodic axis needs >= 3 cells)


def _slab():
    """Periodic-in-x,y slab of lattice fluid, 8 layers thick, free surfaces above and below."""
    n = NS
    c = wl.periodic_cloud("slab", n, DP, 0.0, 5, vel_sigma=0.0, rho_sigma=0.0)
    keep = (c.pos[:, 2] > 1 * DP) & (c.pos[:, 2] < 9 * DP)
    c.pos, c.vel, c.rho, c.ptype = c.pos[keep], c.vel[keep], c.rho[keep], c.ptype[keep]
    c.params["g"] = (0.0, 0.0, 0.0)
    c.params["periodic"] = (1, 1, 0)           # the two free surfaces do not see each other across z
    return c


def _numpy_conc_gradc(p, x, rho, L):
    """Independent brute force: minimum image in x, y over the box length L, plain distances."""
    m = p["rho0"] * DP ** 3
    n = len(x)
    d = x[:, None, :] - x[None, :, :]
    d[:, :, :2] -= L * np.rint(d[:, :, :2] / L)
    r = np.linalg.norm(d, axis=2)
    W = np.zeros_like(r); f = np.zeros_like(r)
    ii, jj = np.nonzero(r < 2 * p["h"])
    W[ii, jj] = [oracle.W(3, p["h"], float(t)) for t in r[ii, jj]]
    f[ii, jj] = [oracle.fab(3, p["h"], float(t)) for t in r[ii, jj]]
    V = m / rho
    conc = (W * V[None, :]).sum(axis=1)                        # self included
    np.fill_diagonal(f, 0.0)
    dC = conc[None, :] - conc[:, None]
    g = ((V[None, :] * dC * f)[:, :, None] * d).sum(axis=1)
    return conc, g


def test_shifting_gradient_at_a_free_surface_against_numpy_bruteforce():
    """grad C_a = sum_b V_b (C_b - C_a) grad_a W_ab (Eq. 53) on a slab with two free surfaces: equal to an independent
    numpy evaluation; points INTO the fluid (towards higher concentration) in the surface layers, so the Fickian shift
    -D_s grad C points out of the fluid there (which is why Eq. 54 exists); zero in x, y by symmetry."""
    c = _slab()
    p = dict(c.params, shift_model=1, shift_coef=2.0)
    cell, u, out = oracle.canonicalize(p, c.pos)
    x = oracle.position(p, cell, u)
    rho = np.full(c.n, 1000.0) + 2.0 * wl.normal01(1, np.arange(c.n), 0)
    conc = oracle.concentration(p, cell, u, out, rho, c.ptype, mode=1)
    vel = np.tile([0.3, 0.0, 0.4], (c.n, 1))
    shift, gradc = oracle.shift_velocity(p, cell, u, out, vel, rho, c.ptype, conc, mode=1)
    L = NS * DP
    conc_np, g_np = _numpy_conc_gradc(p, x, rho, L)
    np.testing.assert_allclose(conc, conc_np, rtol=1e-12)
    np.testing.assert_allclose(gradc, g_np, rtol=1e-9, atol=1e-9 * np.abs(g_np).max())
    top = x[:, 2] > 8 * DP
    bot = x[:, 2] < 2 * DP
    assert np.all(gradc[top, 2] < 0) and np.all(gradc[bot, 2] > 0)          # towards the bulk
    assert np.all(conc[top] < 0.8) and conc[(x[:, 2] > 4 * DP) & (x[:, 2] < 6 * DP)].min() > 0.99
    # Eq. 40-41: delta r / dt = -A_s h |v| grad C
    np.testing.assert_allclose(shift, -2.0 * p["h"] * 0.5 * gradc, rtol=1e-12, atol=1e-18)
    assert np.all(shift[top, 2] > 0)                                        # out of the fluid
    # mode 0 == mode 1
    s0, g0 = oracle.shift_velocity(p, cell, u, out, vel, rho, c.ptype, conc, mode=0)
    np.testing.assert_allclose(g0, gradc, rtol=1e-12, atol=1e-12 * np.abs(gradc).max())


def test_shifting_scales_with_A_s_and_speed_and_the_free_surface_form():
    c = _slab()
    cell, u, out = oracle.canonicalize(c.params, c.pos)
    rho = np.full(c.n, 1000.0)
    speed = 0.1 + wl.uniform01(2, np.arange(c.n), 0)
    vel = np.stack([speed, 0 * speed, 0 * speed], axis=1)
    base = dict(c.params, shift_model=1)
    s2, g = oracle.shift_velocity(dict(base, shift_coef=2.0), cell, u, out, vel, rho, c.ptype, mode=1)
    s6, _ = oracle.shift_velocity(dict(base, shift_coef=6.0), cell, u, out, vel, rho, c.ptype, mode=1)
    np.testing.assert_allclose(s6, 3.0 * s2, rtol=1e-13)                      # linear in A_s (Eq. 41)
    np.testing.assert_allclose(s2, -2.0 * base["h"] * speed[:, None] * g, rtol=1e-13)   # and in |v_a|
    s0, _ = oracle.shift_velocity(dict(base, shift_coef=2.0), cell, u, out, 0 * vel, rho, c.ptype, mode=1)
    assert np.all(s0 == 0.0)
    # Eq. 54 (reading A29): particles with C_a < shift_fs_conc move only along n = -grad C/|grad C| by
    # -D_s a_n (dC/dn - beta_n), dC/dn = -|grad C|; a_n = 0 freezes them; the others keep Eq. 40
    conc = oracle.concentration(base, cell, u, out, rho, c.ptype, mode=1)
    fs = conc < 0.9
    assert 0 < fs.sum() < c.n
    sa, _ = oracle.shift_velocity(dict(base, shift_coef=2.0, shift_fs_conc=0.9), cell, u, out, vel, rho, c.ptype, mode=1)
    assert np.all(sa[fs] == 0.0)
    np.testing.assert_array_equal(sa[~fs], s2[~fs])
    sb, _ = oracle.shift_velocity(dict(base, shift_coef=2.0, shift_fs_conc=0.9, shift_alpha_n=0.1, shift_beta_n=3.0),
                                  cell, u, out, vel, rho, c.ptype, mode=1)
    gn = np.linalg.norm(g, axis=1)
    nvec = -g / gn[:, None]
    want = (-2.0 * base["h"] * speed * 0.1 * (-gn - 3.0))[:, None] * nvec
    np.testing.assert_allclose(sb[fs], want[fs], rtol=1e-12)
    np.testing.assert_array_equal(sb[~fs], s2[~fs])


@pytest.mark.parametrize("scheme", ["symplectic", "verlet"])
def test_shifting_in_the_steppers_moves_positions_by_dt_times_shift(scheme):
    """r^{n+1}(shifting) - r^{n+1}(no shifting) = dt * s, with s the shifting velocity of the state the last pass of
    the step saw: the half-step state of the symplectic scheme (rebuilt here from the pinned interaction pass),
    the state n of the Verlet scheme.  Velocities and densities are not touched by the shift."""
    c = _slab()
    p = dict(c.params, alpha=0.01, delta=0.1)
    vel = 0.2 * np.stack([wl.normal01(4, np.arange(c.n), k) for k in range(3)], axis=1)
    rho = np.full(c.n, 1000.0)
    a = oracle.State(p, c.pos, vel, rho, c.ptype)
    b = oracle.State(dict(p, shift_model=1, shift_coef=2.0), c.pos, vel, rho, c.ptype)
    x0 = a.pos.copy()
    first = a.interactions()
    if scheme == "symplectic":
        a.step(1); b.step(1)
        dt = a.dt_hist[0]
        xh = x0 + 0.5 * dt * vel
        ch, uh, oh = oracle.canonicalize(p, xh)
        vh = vel + 0.5 * dt * first["acc"]
        rh = rho + 0.5 * dt * first["drho"]
        s, _ = oracle.shift_velocity(b.p, ch, uh, oh, vh, rh, c.ptype, mode=1)
    else:
        a.step_verlet(1, 4); b.step_verlet(1, 4)
        dt = a.dt_hist[0]
        s, _ = oracle.shift_velocity(b.p, *oracle.canonicalize(p, x0), vel, rho, c.ptype, mode=1)
    assert b.dt_hist[0] == dt
    q = 2 ** -22 * oracle.grid(p)[0]
    L = NS * DP
    d = b.pos - a.pos
    d[:, :2] -= L * np.rint(d[:, :2] / L)
    assert np.abs(dt * s).max() > 50 * q                         # visible against the position grid
    np.testing.assert_allclose(d, dt * s, rtol=0, atol=1.01 * q)
    np.testing.assert_array_equal(a.vel, b.vel)
    np.testing.assert_array_equal(a.rho, b.rho)


def test_obstacle_normals_geometry():
    """workloads.obstacle_normals (mDBC input of the obstacle dam break): every obstacle particle gets the vector to its
    nearest wetted obstacle face -- one axis only, half a spacing for the outermost layer, never towards the floor the
    obstacle stands on -- so that its ghost node r + 2n is its mirror image outside the obstacle; the tank's own
    particles keep the box_normals vectors."""
    dp = 0.02
    obs = ((15, 6, 0), (5, 8, 6))
    c = wl.dam_break("obstacle", 3, dp, (40, 20, 20), (15, 20, 15), 0.01, 4321, 0.3, obstacle=obs)
    base = wl.dam_break("plain", 3, dp, (40, 20, 20), (15, 20, 15), 0.01, 4321, 0.3)
    o_lo = np.array(obs[0]) * dp
    o_hi = o_lo + np.array(obs[1]) * dp
    rows = np.arange(base.n_bound, c.n_bound)                   # the obstacle's particles follow the tank's
    assert rows.size == 5 * 8 * 6 and (c.ptype[rows] != 0).all()
    np.testing.assert_array_equal(c.normals[:base.n_bound], base.normals[:base.n_bound])
    assert (c.normals[c.ptype == 0] == 0).all()
    nrm, pos = c.normals[rows], c.pos[rows]
    assert ((nrm != 0).sum(axis=1) == 1).all()                  # one face each
    assert (nrm[:, 2] >= 0).all()                               # the bottom face lies on the floor: not an interface
    ghost = pos + 2.0 * nrm
    outside = ((ghost < o_lo) | (ghost > o_hi)).any(axis=1)
    assert outside.all()
    # mirror image: the interface point r + n lies on an obstacle face
    face = pos + nrm
    on_face = (np.abs(face - o_lo) < 1e-12) | (np.abs(face - o_hi) < 1e-12)
    assert (on_face & (nrm != 0)).any(axis=1).all()
    # nearest face: |n| equals the smallest distance to any wetted face (all but z = 0)
    d = np.concatenate([pos - o_lo, o_hi - pos], axis=1)[:, [0, 1, 3, 4, 5]]
    np.testing.assert_allclose(np.abs(nrm).sum(axis=1), d.min(axis=1), rtol=0, atol=1e-15)
    assert np.isclose(np.abs(nrm).sum(axis=1).min(), 0.5 * dp)
    # 2-D: no y component, same rule
    c2 = wl.dam_break("obstacle2d", 2, dp, (60, 1, 30), (20, 1, 20), 0.01, 5, 0.4, obstacle=((30, 0, 0), (4, 1, 6)))
    ob2 = (c2.ptype != 0) & (c2.pos[:, 0] > 0.6) & (c2.pos[:, 0] < 0.68) & (c2.pos[:, 2] > 0) & (c2.pos[:, 2] < 0.12)
    assert ob2.sum() == 24 and (c2.normals[ob2, 1] == 0).all() and ((c2.normals[ob2] != 0).sum(axis=1) == 1).all()
