"""Physics pins for the whole oracle step (SURVEY.md section 8(c), P1, P3, P4, P8-P12 and the
R8 time-step reading).  None of the expected values comes from the oracle or the CUDA path."""
import itertools
import os

import numpy as np
import pytest

import oracle
from oracle import OracleHydro, BC_OUTFLOW, BC_REFLECT, BC_PERIODIC
from paper_1812_07977_b200 import inputs

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _golden(name):
    out = {}
    with open(os.path.join(GOLD, name)) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                k, v = line.split()
                out[k] = float(v)
    return out


def _run(U, gamma, dx, bc, steps, cfl=0.7, theta=None):
    nz, ny, nx = U.shape[1:]
    o = OracleHydro(nx, ny, nz, gamma, dx, bc)
    o.set_cfl(cfl)
    if theta is not None:
        o.set_limiter_theta(theta)
    o.set_state(U)
    for _ in range(steps):
        o.step(o.cfl_dt())
    out = o.get_state()
    o.close()
    return out


# ---------------------------------------------------------------- P1 uniform state

@pytest.mark.parametrize("bc", [(BC_OUTFLOW,) * 6, (BC_PERIODIC,) * 6,
                                (BC_OUTFLOW, BC_OUTFLOW, BC_PERIODIC, BC_PERIODIC,
                                 BC_OUTFLOW, BC_OUTFLOW)])
def test_uniform_state_with_velocity_stays_bit_identical(bc):
    nx, ny, nz = 6, 5, 7
    ones = np.ones((nz, ny, nx))
    U = inputs.conserved_from_primitive(0.7 * ones, 0.31 * ones, -0.17 * ones, 0.53 * ones,
                                        1.3 * ones, 1.4)
    out = _run(U, 1.4, 0.1, bc, 5)
    assert np.array_equal(out, U)


def test_uniform_state_at_rest_with_walls_stays_bit_identical():
    ones = np.ones((5, 6, 4))
    z = 0 * ones
    U = inputs.conserved_from_primitive(0.3 * ones, z, z, z, 2.1 * ones, 5 / 3)
    out = _run(U, 5 / 3, 0.05, (BC_REFLECT,) * 6, 5)
    assert np.array_equal(out, U)


# ---------------------------------------------------------------- P3 conservation (periodic)

def test_periodic_conservation_to_roundoff_config4_shape():
    n = 24
    U = inputs.noise(n, seed=12345)
    steps = 20
    out = _run(U, 5 / 3, 1.0 / n, (BC_PERIODIC,) * 6, steps, cfl=0.5)
    assert not np.array_equal(out, U)
    for v in (0, 4):
        drift = abs(out[v].sum() - U[v].sum()) / abs(U[v].sum())
        assert drift <= 1e-15 * steps, (v, drift)
    mscale = np.abs(U[1:4]).sum()
    for v in (1, 2, 3):
        drift = abs(out[v].sum() - U[v].sum()) / mscale
        assert drift <= 1e-15 * steps, (v, drift)


def test_reflecting_box_conserves_mass_and_energy():
    n = 12
    U = inputs.random_state(n, n, n, seed=3, vamp=0.2)
    out = _run(U, 1.4, 1.0 / n, (BC_REFLECT,) * 6, 10)
    for v in (0, 4):
        assert abs(out[v].sum() - U[v].sum()) <= 1e-14 * abs(U[v].sum())


# ---------------------------------------------------------------- P4 cubic-group symmetry

def test_sphere_keeps_cubic_group_symmetry_bitwise():
    n = 16
    U = inputs.sphere(n)
    out = _run(U, 1.4, 1.0 / n, (BC_OUTFLOW,) * 6, 12)
    assert np.abs(out[1]).max() > 1e-3            # the flow has started
    for perm in itertools.permutations((0, 1, 2)):
        assert np.array_equal(inputs.permute_axes(out, perm), out), perm
    for a in range(3):
        assert np.array_equal(inputs.reflect_axis(out, a), out), a


def test_equivariance_under_axis_permutation_and_reflection_random_state():
    # stronger than P4: arbitrary data, every per-dimension code path must be the same code
    U = inputs.random_state(5, 6, 7, seed=11, vamp=0.4)
    bc = (BC_PERIODIC,) * 6
    ref = _run(U, 1.4, 0.1, bc, 3)
    for perm in itertools.permutations((0, 1, 2)):
        got = _run(inputs.permute_axes(U, perm), 1.4, 0.1, bc, 3)
        assert np.array_equal(got, inputs.permute_axes(ref, perm)), perm
    for a in range(3):
        got = _run(inputs.reflect_axis(U, a), 1.4, 0.1, bc, 3)
        assert np.array_equal(got, inputs.reflect_axis(ref, a)), a


# ---------------------------------------------------------------- P8 translation invariance

def test_periodic_translation_invariance_bitwise():
    U = inputs.random_state(6, 5, 7, seed=21, vamp=0.4)
    bc = (BC_PERIODIC,) * 6
    ref = _run(U, 1.4, 0.1, bc, 3)
    for shift in [(1, 0, 0), (0, 2, 0), (0, 0, 3), (5, 4, 6)]:
        sh = (shift[2], shift[1], shift[0])
        got = _run(np.roll(U, sh, axis=(1, 2, 3)), 1.4, 0.1, bc, 3)
        assert np.array_equal(got, np.roll(ref, sh, axis=(1, 2, 3))), shift


# ---------------------------------------------------------------- P9 wall = mirror image

@pytest.mark.parametrize("axis", [0, 1, 2])
def test_reflecting_wall_equals_mirrored_domain(axis):
    n, m = 6, 4
    shape = [m, m, m]
    shape[axis] = n
    nx, ny, nz = shape
    U = inputs.random_state(nx, ny, nz, seed=31 + axis, vamp=0.3)
    bc = [BC_PERIODIC] * 6
    bc[2 * axis] = BC_REFLECT
    bc[2 * axis + 1] = BC_REFLECT
    steps = 4
    # same dt sequence on both sides: the doubled periodic domain has the same max speed
    got = _run(U, 1.4, 0.1, tuple(bc), steps)
    big = np.concatenate([U, inputs.reflect_axis(U, axis)], axis=3 - axis)
    ref = _run(big, 1.4, 0.1, (BC_PERIODIC,) * 6, steps)
    sl = [slice(None)] * 4
    sl[3 - axis] = slice(0, n)
    assert np.array_equal(got, ref[tuple(sl)])


# ---------------------------------------------------------------- P10 axis relabelling of the Sod tube

def test_sod_tube_along_y_and_z_equals_x_run_bitwise():
    nx = 32
    U = inputs.sod(nx, 4, 4)
    bcx = (BC_OUTFLOW, BC_OUTFLOW, BC_PERIODIC, BC_PERIODIC, BC_PERIODIC, BC_PERIODIC)
    ref = _run(U, 1.4, 1.0 / nx, bcx, 15)
    # every transverse row is identical and transverse momenta vanish exactly (P2 addendum)
    assert np.array_equal(ref, np.broadcast_to(ref[:, :1, :1, :], ref.shape))
    assert not ref[2].any() and not ref[3].any()
    for perm in [(1, 2, 0), (2, 0, 1), (1, 0, 2)]:
        # new axis a is old axis perm[a]; old x (the tube) becomes new axis perm.index(0)
        Up = inputs.permute_axes(U, perm)
        bc = [0] * 6
        for a in range(3):
            bc[2 * a], bc[2 * a + 1] = bcx[2 * perm[a]], bcx[2 * perm[a] + 1]
        got = _run(Up, 1.4, 1.0 / nx, tuple(bc), 15)
        assert np.array_equal(got, inputs.permute_axes(ref, perm)), perm


# ---------------------------------------------------------------- P11 / R8 time step

def test_first_time_step_of_config0_matches_hand_value():
    c = inputs.config(0)
    o = OracleHydro(*c.shape, c.gamma, c.dx, c.bc)
    o.set_cfl(c.cfl)
    o.set_state(c.state())
    assert o.max_signal_speed() == np.sqrt(1.4)
    gold = _golden("cfg0_first_dt.txt")["dt0"]
    assert abs(o.cfl_dt() - gold) <= 1e-12 * gold
    assert o.cfl_dt() == (0.7 / 3.0) * ((1.0 / 32.0) / np.sqrt(1.4))


def test_cfl_uses_euclidean_speed_plus_sound_speed():
    g = 1.4
    ones = np.ones((4, 4, 4))
    U = inputs.conserved_from_primitive(ones, 3 * ones, 4 * ones, 12 * ones, g ** -1 * ones, g)
    o = OracleHydro(4, 4, 4, g, 0.5, (BC_PERIODIC,) * 6)
    o.set_state(U)
    assert abs(o.max_signal_speed() - 14.0) <= 1e-14 * 14      # |v| = 13, c = 1
    o.set_cfl(0.6)
    assert abs(o.cfl_dt() - 0.2 * 0.5 / 14.0) <= 1e-16


def test_literal_cfl_reading_goes_unphysical_on_config0_R8():
    """DESIGN.md R8: dt = CFL*min(dx/(|v|+c)) without the /3 gives negative pressure in config 0,
    while the adopted reading keeps rho >= 0.125 and p > 0."""
    c = inputs.config(0)
    o = OracleHydro(*c.shape, c.gamma, c.dx, c.bc)
    U0 = c.state()
    o.set_state(U0)
    o.step(c.cfl * c.dx / o.max_signal_speed())
    with pytest.raises(oracle.OracleError) as e:
        for _ in range(3):
            o.step(c.cfl * c.dx / o.max_signal_speed())
    assert e.value.code == 4


def test_unphysical_state_is_reported():
    U = inputs.random_state(4, 4, 4)
    U[0, 1, 2, 3] = -1.0
    o = OracleHydro(4, 4, 4, 1.4, 0.1, (BC_PERIODIC,) * 6)
    o.set_state(U)
    with pytest.raises(oracle.OracleError) as e:
        o.cfl_dt()
    assert e.value.code == 4


# ---------------------------------------------------------------- P12 third opinion, config 0

def test_config0_matches_survey_probe_values():
    c = inputs.config(0)
    gold = _golden("cfg0_survey_probe.txt")
    o = OracleHydro(*c.shape, c.gamma, c.dx, c.bc)
    o.set_cfl(c.cfl)
    o.set_state(c.state())
    for _ in range(c.steps):
        dt = o.cfl_dt()
        o.step(dt)
    U = o.get_state()
    dx3 = c.dx ** 3
    rel = lambda a, b: abs(a - b) / abs(b)
    assert rel(dt, gold["dt_step20"]) < 1e-11
    assert rel(U[0].sum() * dx3, gold["mass"]) < 1e-11
    assert rel(U[4].sum() * dx3, gold["energy"]) < 1e-11
    cell = U[:, 16, 16, 16]
    assert rel(cell[0], gold["rho_16_16_16"]) < 1e-11
    assert rel(cell[1], gold["mx_16_16_16"]) < 1e-9 and cell[1] == cell[2] == cell[3]
    assert rel(cell[4], gold["E_16_16_16"]) < 1e-11
    cell = U[:, 16, 16, 24]
    assert rel(cell[0], gold["rho_24_16_16"]) < 1e-11
    assert rel(cell[1], gold["mx_24_16_16"]) < 1e-11
    assert rel(cell[2], gold["my_24_16_16"]) < 1e-10 and cell[2] == cell[3]
    assert rel(cell[4], gold["E_24_16_16"]) < 1e-11
    assert rel(np.abs(U[1] / U[0]).max(), gold["max_abs_vx"]) < 1e-11
    assert U[0].min() == gold["min_rho"]


# ---------------------------------------------------------------- evolve (O8, R14)

def test_evolve_lands_exactly_on_t_final_and_matches_manual_loop():
    U = inputs.sod(32, 4, 4)
    bc = (BC_OUTFLOW, BC_OUTFLOW, BC_PERIODIC, BC_PERIODIC, BC_PERIODIC, BC_PERIODIC)
    a = OracleHydro(32, 4, 4, 1.4, 1 / 32, bc)
    a.set_state(U)
    n = a.evolve(0.05)
    t, steps = a.get_time()
    assert t == 0.05 and steps == n
    b = OracleHydro(32, 4, 4, 1.4, 1 / 32, bc)
    b.set_state(U)
    tt, k = 0.0, 0
    while tt < 0.05:
        dt = b.cfl_dt()
        if tt + dt >= 0.05:
            dt = 0.05 - tt
            tt = 0.05
        else:
            tt = tt + dt
        b.step(dt)
        k += 1
    assert k == n
    assert np.array_equal(a.get_state(), b.get_state())


def test_thread_count_does_not_change_results():
    U = inputs.random_state(9, 7, 8, seed=5)
    nth = oracle.get_threads()
    try:
        oracle.set_threads(1)
        a = _run(U, 1.4, 0.1, (BC_OUTFLOW,) * 6, 3)
        oracle.set_threads(max(2, nth))
        b = _run(U, 1.4, 0.1, (BC_OUTFLOW,) * 6, 3)
    finally:
        oracle.set_threads(nth)
    assert np.array_equal(a, b)
