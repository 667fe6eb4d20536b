"""Pins for the oracle's building blocks: sum3 (R17), limiter (P6), HLL (P7), primitive
recovery (O2), ghost fill (O1).  Expected values come from closed forms and special cases,
not from the oracle itself."""
import itertools
import math

import numpy as np
import pytest

import oracle
from oracle import OracleHydro, BC_OUTFLOW, BC_REFLECT, BC_PERIODIC
from paper_1812_07977_b200 import inputs


# ---------------------------------------------------------------- sum3 (R17)

def test_sum3_is_permutation_symmetric_and_close_to_exact():
    rng = np.random.default_rng(1)
    for _ in range(200):
        a, b, c = (rng.uniform(-1, 1, 3) * 10.0 ** rng.integers(-8, 8, 3)).tolist()
        vals = {oracle.sum3(*p) for p in itertools.permutations((a, b, c))}
        assert len(vals) == 1
        s = vals.pop()
        assert abs(s - math.fsum((a, b, c))) <= 2 * np.spacing(abs(a) + abs(b) + abs(c))


def test_sum3_exact_cases():
    assert oracle.sum3(1.0, 2.0, 3.0) == 6.0
    assert oracle.sum3(0.0, 0.0, 0.0) == 0.0
    assert oracle.sum3(-5.0, 5.0, 1e-30) == 1e-30      # (smallest + largest) first
    assert oracle.sum3(7.0, -7.0, 0.0) == 0.0


# ---------------------------------------------------------------- limiter (P6)

def test_minmod_theta1_is_classical_minmod():
    rng = np.random.default_rng(2)
    for _ in range(500):
        a, b = rng.normal(size=2).tolist()
        want = 0.0 if a * b <= 0 else math.copysign(min(abs(a), abs(b)), a)
        assert oracle.minmod(1.0, a, b) == want


def test_minmod_theta2_is_mc_limiter():
    rng = np.random.default_rng(3)
    for _ in range(500):
        a, b = rng.normal(size=2).tolist()
        want = 0.0 if a * b <= 0 else math.copysign(
            min(2 * abs(a), 2 * abs(b), 0.5 * abs(a + b)), a)
        assert oracle.minmod(2.0, a, b) == want


def test_minmod_sign_cases_and_extrema():
    th = 1.4
    assert oracle.minmod(th, 0.0, 1.0) == 0.0
    assert oracle.minmod(th, 1.0, 0.0) == 0.0
    assert oracle.minmod(th, 0.0, 0.0) == 0.0
    assert oracle.minmod(th, 1.0, -1.0) == 0.0          # extremum, a = -b
    assert oracle.minmod(th, -2.0, 3.0) == 0.0
    # smooth region: central slope is the smallest argument
    assert oracle.minmod(th, 1.0, 1.0) == 1.0
    assert oracle.minmod(th, -1.0, -1.0) == -1.0
    # steep side: theta * smaller difference limits
    assert oracle.minmod(th, 1.0, 10.0) == 1.4
    assert oracle.minmod(th, 10.0, 1.0) == 1.4
    assert oracle.minmod(th, -1.0, -10.0) == -1.4
    # central branch: a=1, b=2 -> min(1.4, 2.8, 1.5) = 1.4 ; a=1, b=1.5 -> min(1.4, 2.1, 1.25)
    assert oracle.minmod(th, 1.0, 1.5) == 1.25
    assert oracle.minmod(th, -1.0, -1.5) == -1.25


def test_minmod_symmetry_homogeneity_and_bound():
    rng = np.random.default_rng(4)
    for _ in range(300):
        a, b = rng.normal(size=2).tolist()
        th = float(rng.uniform(1, 2))
        m = oracle.minmod(th, a, b)
        assert oracle.minmod(th, b, a) == m                     # argument swap
        assert oracle.minmod(th, -a, -b) == -m                  # odd
        assert oracle.minmod(th, 4.0 * a, 4.0 * b) == 4.0 * m   # power-of-two scaling exact
        assert abs(m) <= th * min(abs(a), abs(b)) + 1e-300
        assert abs(m) <= 0.5 * abs(a + b) + 1e-300


# ---------------------------------------------------------------- primitive recovery (O2)

def test_primitive_roundtrip_against_definition():
    g = 1.4
    rho, vx, vy, vz, p = 0.7, 0.3, -0.2, 0.9, 1.3
    E = p / (g - 1) + 0.5 * rho * (vx * vx + vy * vy + vz * vz)
    W = oracle.primitive(g, [rho, rho * vx, rho * vy, rho * vz, E])
    np.testing.assert_allclose(W, [rho, vx, vy, vz, p], rtol=4e-16, atol=0)
    # at rest with power-of-two data the recovery is exact
    W = oracle.primitive(1.5, [0.5, 0.0, 0.0, 0.0, 4.0])
    assert W.tolist() == [0.5, 0.0, 0.0, 0.0, 2.0]


# ---------------------------------------------------------------- HLL (P7)

def _phys_flux(W, d, g):
    rho, v, p = W[0], W[1:4], W[4]
    E = p / (g - 1) + 0.5 * rho * float(np.dot(v, v))
    F = np.array([rho * v[d], rho * v[0] * v[d], rho * v[1] * v[d], rho * v[2] * v[d],
                  (E + p) * v[d]])
    F[1 + d] += p
    U = np.array([rho, rho * v[0], rho * v[1], rho * v[2], E])
    return F, U


@pytest.mark.parametrize("d", [0, 1, 2])
def test_hll_consistency_equal_states_give_physical_flux(d):
    rng = np.random.default_rng(10 + d)
    g = 1.4
    for _ in range(100):
        W = np.array([rng.uniform(0.2, 2), *rng.uniform(-2, 2, 3), rng.uniform(0.2, 2)])
        F = oracle.hll_flux(g, d, W, W)
        Fx, _ = _phys_flux(W, d, g)
        scale = np.abs(Fx).max()
        assert np.abs(F - Fx).max() <= 8e-16 * scale


@pytest.mark.parametrize("d", [0, 1, 2])
def test_hll_supersonic_upwinding(d):
    g = 1.4
    WL = np.array([1.0, 0.1, -0.2, 0.3, 1.0]); WR = np.array([0.6, -0.1, 0.25, 0.1, 0.7])
    WL[1 + d] = 5.0; WR[1 + d] = 4.0               # both v_n - c > 0  ->  F = F_L
    F = oracle.hll_flux(g, d, WL, WR)
    FL, _ = _phys_flux(WL, d, g)
    np.testing.assert_allclose(F, FL, rtol=5e-16, atol=0)
    WL[1 + d] = -5.0; WR[1 + d] = -4.0             # both v_n + c < 0  ->  F = F_R
    F = oracle.hll_flux(g, d, WL, WR)
    FR, _ = _phys_flux(WR, d, g)
    np.testing.assert_allclose(F, FR, rtol=5e-16, atol=0)


@pytest.mark.parametrize("d", [0, 1, 2])
def test_hll_at_rest_equal_sound_speed_is_rusanov_form(d):
    # c_L = c_R = c with different densities: F = (F_L+F_R)/2 - c (U_R-U_L)/2
    g = 1.4
    WL = np.array([1.0, 0, 0, 0, 1.0]); WR = np.array([0.25, 0, 0, 0, 0.25])
    c = math.sqrt(g)
    FL, UL = _phys_flux(WL, d, g); FR, UR = _phys_flux(WR, d, g)
    want = 0.5 * (FL + FR) - 0.5 * c * (UR - UL)
    F = oracle.hll_flux(g, d, WL, WR)
    np.testing.assert_allclose(F, want, rtol=4e-16, atol=1e-17)


@pytest.mark.parametrize("d", [0, 1, 2])
def test_hll_mirror_antisymmetry_is_exact(d):
    rng = np.random.default_rng(20 + d)
    g = 5.0 / 3.0
    for _ in range(100):
        WL = np.array([rng.uniform(0.2, 2), *rng.uniform(-2, 2, 3), rng.uniform(0.2, 2)])
        WR = np.array([rng.uniform(0.2, 2), *rng.uniform(-2, 2, 3), rng.uniform(0.2, 2)])
        F = oracle.hll_flux(g, d, WL, WR)
        ML, MR = WR.copy(), WL.copy()              # mirrored problem: swap sides, flip v_n
        ML[1 + d] = -ML[1 + d]; MR[1 + d] = -MR[1 + d]
        G = oracle.hll_flux(g, d, ML, MR)
        want = -F
        want[1 + d] = F[1 + d]                     # normal-momentum flux is even
        assert np.array_equal(G, want)


def test_hll_axis_relabelling_is_exact():
    rng = np.random.default_rng(30)
    g = 1.4
    for _ in range(50):
        WL = np.array([rng.uniform(0.2, 2), *rng.uniform(-2, 2, 3), rng.uniform(0.2, 2)])
        WR = np.array([rng.uniform(0.2, 2), *rng.uniform(-2, 2, 3), rng.uniform(0.2, 2)])
        Fx = oracle.hll_flux(g, 0, WL, WR)
        # relabel so that old x becomes new y: velocities (vx,vy,vz) -> (vz,vx,vy)
        perm = [0, 3, 1, 2, 4]
        Fy = oracle.hll_flux(g, 1, WL[perm], WR[perm])
        assert np.array_equal(Fy, Fx[perm])


# ---------------------------------------------------------------- ghost fill (O1, R9)

def _filled(bc, nx=3, ny=4, nz=5, seed=5):
    U = inputs.random_state(nx, ny, nz, seed=seed)
    o = OracleHydro(nx, ny, nz, 1.4, 0.1, bc)
    o.set_state(U)
    o.ghost_fill()
    return U, o.get_padded()


def test_ghost_fill_outflow():
    U, P = _filled((BC_OUTFLOW,) * 6)
    nx, ny, nz = 3, 4, 5
    act = P[:, 2:-2, 2:-2, 2:-2]
    assert np.array_equal(act, U)
    for g in (0, 1):
        assert np.array_equal(P[:, 2:-2, 2:-2, g], U[:, :, :, 0])
        assert np.array_equal(P[:, 2:-2, 2:-2, nx + 2 + g], U[:, :, :, -1])
        assert np.array_equal(P[:, 2:-2, g, 2:-2], U[:, :, 0, :])
        assert np.array_equal(P[:, 2:-2, ny + 2 + g, 2:-2], U[:, :, -1, :])
        assert np.array_equal(P[:, g, 2:-2, 2:-2], U[:, 0, :, :])
        assert np.array_equal(P[:, nz + 2 + g, 2:-2, 2:-2], U[:, -1, :, :])


def test_ghost_fill_periodic():
    U, P = _filled((BC_PERIODIC,) * 6)
    nx, ny, nz = 3, 4, 5
    for g in (0, 1):
        assert np.array_equal(P[:, 2:-2, 2:-2, g], U[:, :, :, nx - 2 + g])
        assert np.array_equal(P[:, 2:-2, 2:-2, nx + 2 + g], U[:, :, :, g])
        assert np.array_equal(P[:, 2:-2, g, 2:-2], U[:, :, ny - 2 + g, :])
        assert np.array_equal(P[:, 2:-2, ny + 2 + g, 2:-2], U[:, :, g, :])
        assert np.array_equal(P[:, g, 2:-2, 2:-2], U[:, nz - 2 + g, :, :])
        assert np.array_equal(P[:, nz + 2 + g, 2:-2, 2:-2], U[:, g, :, :])


def test_ghost_fill_reflecting():
    U, P = _filled((BC_REFLECT,) * 6)
    nx, ny, nz = 3, 4, 5
    sx = np.array([1, -1, 1, 1, 1.0])[:, None, None]
    sy = np.array([1, 1, -1, 1, 1.0])[:, None, None]
    sz = np.array([1, 1, 1, -1, 1.0])[:, None, None]
    # ghost at distance g+1 outside the wall mirrors the active cell at distance g+1 inside
    assert np.array_equal(P[:, 2:-2, 2:-2, 1], sx * U[:, :, :, 0])
    assert np.array_equal(P[:, 2:-2, 2:-2, 0], sx * U[:, :, :, 1])
    assert np.array_equal(P[:, 2:-2, 2:-2, nx + 2], sx * U[:, :, :, -1])
    assert np.array_equal(P[:, 2:-2, 2:-2, nx + 3], sx * U[:, :, :, -2])
    assert np.array_equal(P[:, 2:-2, 1, 2:-2], sy * U[:, :, 0, :])
    assert np.array_equal(P[:, 2:-2, 0, 2:-2], sy * U[:, :, 1, :])
    assert np.array_equal(P[:, 2:-2, ny + 2, 2:-2], sy * U[:, :, -1, :])
    assert np.array_equal(P[:, 2:-2, ny + 3, 2:-2], sy * U[:, :, -2, :])
    assert np.array_equal(P[:, 1, 2:-2, 2:-2], sz * U[:, 0, :, :])
    assert np.array_equal(P[:, 0, 2:-2, 2:-2], sz * U[:, 1, :, :])
    assert np.array_equal(P[:, nz + 2, 2:-2, 2:-2], sz * U[:, -1, :, :])
    assert np.array_equal(P[:, nz + 3, 2:-2, 2:-2], sz * U[:, -2, :, :])


def test_ghost_fill_mixed_faces():
    bc = (BC_OUTFLOW, BC_REFLECT, BC_PERIODIC, BC_PERIODIC, BC_REFLECT, BC_OUTFLOW)
    U, P = _filled(bc)
    nx, ny, nz = 3, 4, 5
    sx = np.array([1, -1, 1, 1, 1.0])[:, None, None]
    sz = np.array([1, 1, 1, -1, 1.0])[:, None, None]
    assert np.array_equal(P[:, 2:-2, 2:-2, 0], U[:, :, :, 0])
    assert np.array_equal(P[:, 2:-2, 2:-2, nx + 3], sx * U[:, :, :, -2])
    assert np.array_equal(P[:, 2:-2, 0, 2:-2], U[:, :, ny - 2, :])
    assert np.array_equal(P[:, 0, 2:-2, 2:-2], sz * U[:, 1, :, :])
    assert np.array_equal(P[:, nz + 3, 2:-2, 2:-2], U[:, -1, :, :])


# ---------------------------------------------------------------- argument checking

def test_create_rejects_bad_arguments():
    ok = (0,) * 6
    for args in [(1, 4, 4, 1.4, 0.1, ok), (4, 4, 4, 1.0, 0.1, ok), (4, 4, 4, 1.4, 0.0, ok),
                 (4, 4, 4, 1.4, 0.1, (0, 0, 0, 0, 0, 3)),
                 (4, 4, 4, 1.4, 0.1, (2, 0, 0, 0, 0, 0))]:
        with pytest.raises(oracle.OracleError):
            OracleHydro(*args)
    o = OracleHydro(4, 4, 4, 1.4, 0.1, ok)
    with pytest.raises(oracle.OracleError) as e:
        o.step(0.1)
    assert e.value.code == 5                      # ERR_NOSTATE
    o.set_state(inputs.random_state(4, 4, 4))
    with pytest.raises(oracle.OracleError):
        o.step(-1.0)
    with pytest.raises(oracle.OracleError):
        o.set_limiter_theta(2.5)
