"""Pins of the oracle's 1D / 2D runs and non-cubic cells (SURVEY.md section 8(f) NEXT-3,
DESIGN.md readings R21-R24; the RiemannProblem runs in 1D, 2D and 3D).

N2 true-1D Sod: L1 convergence to the exact Riemann solution (tests/exact_riemann.py);
N3 2D: x<->y relabelling and both reflections bitwise on a cylindrical Riemann problem;
N4 a 2D run equals the 3D run of the same data made uniform and periodic in z, at equal dt, bitwise;
N5 a 1D run equals the 2D run of y-uniform data at equal dt, bitwise;
N6 anisotropic cells: one RK2 step of single cells against a scalar hand expansion with
   per-axis edges (bitwise), a y-aligned tube on stretched cells against the 1D run (roundoff),
   relabelling of unequal axes (roundoff);
N7 the time-step formula: (CFL/ndim) * min_d(dx_d) / max(|v|+c_s).
The 3D cubic path is pinned separately (tests/test_oracle_digest.py and P1-P12)."""
import math

import numpy as np
import pytest

import exact_riemann as er
import oracle
from oracle import OracleHydro, OracleError
from paper_1812_07977_b200 import inputs
from test_oracle_bruteforce import Grid, hll, prim, s3, slope

OUT, REF, PER = 0, 1, 2
SOD = (1.0, 0.0, 1.0, 0.125, 0.0, 0.1, 1.4)


def make(shape, ndim, dxyz, bc, gamma=1.4, cfl=0.7, theta=None):
    nx, ny, nz = shape
    o = OracleHydro(nx, ny, nz, gamma, dxyz[0], bc, ndim=ndim, dxyz=dxyz)
    o.set_cfl(cfl)
    if theta is not None:
        o.set_limiter_theta(theta)
    return o


# ---------------------------------------------------------------- argument rules, layout

def test_create_nd_argument_rules_and_padded_layout():
    bc = (OUT,) * 6
    for bad in (dict(shape=(8, 2, 1), ndim=1), dict(shape=(8, 1, 2), ndim=2), dict(shape=(1, 1, 1), ndim=1),
                dict(shape=(8, 8, 8), ndim=4), dict(shape=(8, 8, 8), ndim=0)):
        with pytest.raises(OracleError):
            make(bad["shape"], bad["ndim"], (0.1, 0.1, 0.1), bc)
    with pytest.raises(OracleError):
        make((8, 8, 1), 2, (0.1, -0.1, 0.1), bc)
    with pytest.raises(OracleError):
        make((8, 8, 1), 2, (0.1, 0.1, 0.1), (OUT, OUT, PER, OUT, OUT, OUT))
    # entries of inactive axes are ignored
    o = make((6, 5, 1), 2, (0.1, 0.2, -1.0), (OUT, REF, PER, PER, 7, 7))
    assert o.padded_shape == (5, 1, 9, 10)
    U = inputs.random_state(6, 5, 1, seed=4)
    o.set_state(U)
    assert np.array_equal(o.get_state(), U)
    o.ghost_fill()
    P = o.get_padded()
    assert np.array_equal(P[:, 0, 2:7, 2:8], U[:, 0])
    assert np.array_equal(P[:, 0, 2:7, 0], U[:, 0, :, 0]) and np.array_equal(P[:, 0, 2:7, 1], U[:, 0, :, 0])
    m = np.array([1.0, -1.0, 1.0, 1.0, 1.0])[:, None]
    assert np.array_equal(P[:, 0, 2:7, 8], m * U[:, 0, :, 5]) and np.array_equal(P[:, 0, 2:7, 9], m * U[:, 0, :, 4])
    assert np.array_equal(P[:, 0, 0, 2:8], U[:, 0, 3]) and np.array_equal(P[:, 0, 8, 2:8], U[:, 0, 1])


# ---------------------------------------------------------------- N7 time step

@pytest.mark.parametrize("ndim,shape,dxyz", [(1, (9, 1, 1), (0.3, 9.0, 9.0)), (2, (5, 4, 1), (0.3, 0.11, 9.0)),
                                            (3, (4, 3, 5), (0.3, 0.11, 0.2)), (3, (4, 3, 5), (0.07, 0.11, 0.2))])
def test_time_step_formula(ndim, shape, dxyz):
    g, cfl = 5.0 / 3.0, 0.5
    U0 = inputs.random_state(*shape, gamma=g, seed=17)
    o = make(shape, ndim, dxyz, (PER,) * 6, gamma=g, cfl=cfl)
    o.set_state(U0)
    smax = 0.0
    for U in U0.reshape(5, -1).T.tolist():
        inv = 1.0 / U[0]
        vx, vy, vz = U[1] * inv, U[2] * inv, U[3] * inv
        q = s3(vx * vx, vy * vy, vz * vz)
        p = (g - 1.0) * (U[4] - (0.5 * U[0]) * q)
        smax = max(smax, math.sqrt(q) + math.sqrt((g * p) * inv))
    assert o.max_signal_speed() == smax
    assert o.cfl_dt() == (cfl / float(ndim)) * (min(dxyz[:ndim]) / smax)


# ---------------------------------------------------------------- N2 true-1D Sod

def _sod_1d(nx, t_final=0.2):
    o = make((nx, 1, 1), 1, (1.0 / nx,) * 3, (OUT,) * 6)
    o.set_state(inputs.sod(nx, 1, 1))
    n = o.evolve(t_final)
    U = o.get_state()
    assert o.get_time()[0] == t_final and not U[2].any() and not U[3].any()
    x = (np.arange(nx) + 0.5) / nx
    rho_e, u_e, p_e = er.sample((x - 0.5) / t_final, *SOD)
    rho = U[0, 0, 0]
    u = U[1, 0, 0] / rho
    p = 0.4 * (U[4, 0, 0] - 0.5 * rho * u * u)
    return np.abs(rho - rho_e).sum() / nx, np.abs(u - u_e).sum() / nx, np.abs(p - p_e).sum() / nx, n


def test_true_1d_sod_converges_in_l1_to_the_exact_solution():
    nth = oracle.get_threads()
    oracle.set_threads(1)
    try:
        res = {nx: _sod_1d(nx) for nx in (64, 128, 256, 512, 1024)}
    finally:
        oracle.set_threads(nth)
    for a, b in ((64, 128), (128, 256), (256, 512), (512, 1024)):
        for q, need in ((0, 1.6), (1, 1.5), (2, 1.6)):
            assert res[a][q] / res[b][q] >= need, (a, b, q, res[a][q], res[b][q])
    # Courant divisor 1 instead of 3: a third of the embedded run's ~960 steps, similar error level
    assert 300 <= res[512][3] <= 340
    assert res[512][0] < 1.6e-3 and res[512][2] < 1.2e-3      # embedded 3D run: 1.31e-3, 8.6e-4


# ---------------------------------------------------------------- N3 2D symmetry

def _cylinder(n):
    a = 2 * np.arange(n, dtype=np.int64) + 1 - n
    inside = 4 * (a[:, None] ** 2 + a[None, :] ** 2) < n * n
    rho = np.where(inside, 1.0, 0.125)[None]
    p = np.where(inside, 1.0, 0.1)[None]
    z = np.zeros_like(rho)
    return inputs.conserved_from_primitive(rho, z, z, z, p, 1.4)


def test_2d_cylinder_keeps_the_square_symmetries_bitwise():
    n = 24
    o = make((n, n, 1), 2, (1.0 / n,) * 3, (OUT,) * 6)
    o.set_state(_cylinder(n))
    for _ in range(12):
        o.step(o.cfl_dt())
    U = o.get_state()
    assert np.abs(U[1]).max() > 0.05 and not U[3].any()
    T = np.ascontiguousarray(np.transpose(U, (0, 1, 3, 2)))[[0, 2, 1, 3, 4]]      # x <-> y
    assert np.array_equal(T, U)
    for ax, comp in ((3, 1), (2, 2)):                                             # mirror x, mirror y
        M = np.flip(U, axis=ax).copy()
        M[comp] = -M[comp]
        assert np.array_equal(M, U)


# ---------------------------------------------------------------- N4 / N5 embedding

@pytest.mark.parametrize("bcxy", [(PER, PER, PER, PER), (OUT, REF, REF, OUT)])
def test_2d_run_equals_3d_run_of_z_uniform_data_at_equal_dt(bcxy):
    nx, ny, g = 11, 7, 1.4
    U2 = inputs.random_state(nx, ny, 1, gamma=g, seed=8, vamp=0.5)       # v_z != 0 is carried along
    U3 = np.ascontiguousarray(np.repeat(U2, 3, axis=1))
    d = (0.05, 0.05, 0.05)
    o2 = make((nx, ny, 1), 2, d, bcxy + (OUT, OUT), gamma=g)
    o3 = make((nx, ny, 3), 3, d, bcxy + (PER, PER), gamma=g)
    o2.set_state(U2); o3.set_state(U3)
    for _ in range(4):
        dt = o3.cfl_dt()
        assert o2.cfl_dt() == 1.5 * dt or abs(o2.cfl_dt() - 1.5 * dt) <= 4e-16 * dt   # CFL/2 vs CFL/3
        o2.step(dt); o3.step(dt)
    a, b = o2.get_state(), o3.get_state()
    for k in range(3):
        assert np.array_equal(b[:, k], a[:, 0])


def test_1d_run_equals_2d_run_of_y_uniform_data_at_equal_dt():
    nx, g = 23, 5.0 / 3.0
    U1 = inputs.random_state(nx, 1, 1, gamma=g, seed=5, vamp=0.5)
    U2 = np.ascontiguousarray(np.repeat(U1, 4, axis=2))
    o1 = make((nx, 1, 1), 1, (0.1, 0.1, 0.1), (REF, OUT) + (OUT,) * 4, gamma=g)
    o2 = make((nx, 4, 1), 2, (0.1, 0.37, 0.1), (REF, OUT, PER, PER, OUT, OUT), gamma=g)
    o1.set_state(U1); o2.set_state(U2)
    for _ in range(5):
        dt = o2.cfl_dt()
        o1.step(dt); o2.step(dt)
    a, b = o1.get_state(), o2.get_state()
    for j in range(4):
        assert np.array_equal(b[:, 0, j], a[:, 0, 0])


# ---------------------------------------------------------------- N6 anisotropic cells

def _delta_U(grid, idx, g, r, ndim, ry, rz):
    dF = []
    for d in range(ndim):
        def W(o):
            j = list(idx)
            j[d] += o
            return prim(grid.U(j), g)
        Wm2, Wm1, W0, Wp1, Wp2 = W(-2), W(-1), W(0), W(1), W(2)
        sm1 = [slope(Wm2[v], Wm1[v], W0[v]) for v in range(5)]
        s0 = [slope(Wm1[v], W0[v], Wp1[v]) for v in range(5)]
        sp1 = [slope(W0[v], Wp1[v], Wp2[v]) for v in range(5)]
        Fm = hll([Wm1[v] + 0.5 * sm1[v] for v in range(5)], [W0[v] - 0.5 * s0[v] for v in range(5)], d, g)
        Fp = hll([W0[v] + 0.5 * s0[v] for v in range(5)], [Wp1[v] - 0.5 * sp1[v] for v in range(5)], d, g)
        dF.append([Fp[v] - Fm[v] for v in range(5)])
    out = []
    for v in range(5):
        D = dF[0][v]
        if ndim == 2:
            D = D + ry * dF[1][v]
        elif ndim == 3:
            D = s3(D, ry * dF[1][v], rz * dF[2][v])
        out.append(-(r * D))
    return out


def _rk2_cell(U0arr, n, bc, g, dt, dxyz, ndim, idx):
    r, ry, rz = dt / dxyz[0], dxyz[0] / dxyz[1], dxyz[0] / dxyz[2]
    g0 = Grid(lambda j: tuple(U0arr[:, j[2], j[1], j[0]].tolist()), n, bc)
    memo = {}

    def U1(j):
        if j not in memo:
            u0 = g0.U(j)
            du = _delta_U(g0, j, g, r, ndim, ry, rz)
            memo[j] = tuple(u0[v] + du[v] for v in range(5))
        return memo[j]

    g1 = Grid(U1, n, bc)
    u0, u1 = g0.U(idx), U1(tuple(idx))
    du = _delta_U(g1, idx, g, r, ndim, ry, rz)
    return [0.5 * ((u0[v] + u1[v]) + du[v]) for v in range(5)]


@pytest.mark.parametrize("ndim,n,dxyz,bc", [
    (3, (4, 5, 3), (0.1, 0.07, 0.23), (OUT, REF, PER, PER, REF, OUT)),
    (3, (3, 4, 4), (0.2, 0.2, 0.05), (PER,) * 6),
    (2, (5, 4, 1), (0.1, 0.31, 1.0), (REF, OUT, PER, PER, OUT, OUT)),
    (2, (4, 6, 1), (0.3, 0.1, 1.0), (OUT, OUT, REF, REF, OUT, OUT)),
    (1, (7, 1, 1), (0.13, 1.0, 1.0), (REF, OUT, OUT, OUT, OUT, OUT)),
    (1, (2, 1, 1), (0.13, 1.0, 1.0), (PER, PER, OUT, OUT, OUT, OUT)),
])
def test_single_cell_rk2_update_with_per_axis_edges_matches_hand_expansion_bitwise(ndim, n, dxyz, bc):
    g = 1.4
    U0 = inputs.random_state(*n, gamma=g, seed=sum(n) + ndim, vamp=0.6)
    o = make(n, ndim, dxyz, bc, gamma=g)
    o.set_state(U0)
    dt = o.cfl_dt()
    o.step(dt)
    got = o.get_state()
    nx, ny, nz = n
    cells = {(0, 0, 0), (nx - 1, ny - 1, nz - 1), (nx // 2, ny // 2, nz // 2), (nx - 1, 0, 0), (0, ny - 1, nz - 1)}
    for idx in sorted(cells):
        want = _rk2_cell(U0, n, bc, g, dt, dxyz, ndim, idx)
        assert got[:, idx[2], idx[1], idx[0]].tolist() == want, idx


def test_tube_along_y_on_stretched_cells_equals_the_1d_run_to_roundoff():
    """2D grid, data uniform in x, Sod along y with dy = 1/ny and dx = 7.3: the y terms enter the
    update through (dt/dx) * ((dx/dy) * dFy), which must act like dt/dy of the 1D run."""
    ny = 48
    U1 = inputs.sod(ny, 1, 1)                                           # along x
    U2 = np.zeros((5, 1, ny, 3))
    U2[[0, 2, 4]] = U1[[0, 1, 4], 0, 0][:, None, :, None]               # along y: m_y <- m_x
    o1 = make((ny, 1, 1), 1, (1.0 / ny, 1.0, 1.0), (OUT,) * 6)
    o2 = make((3, ny, 1), 2, (7.3, 1.0 / ny, 1.0), (PER, PER, OUT, OUT, OUT, OUT))
    o1.set_state(U1); o2.set_state(U2)
    for _ in range(20):
        dt = o1.cfl_dt()
        o1.step(dt); o2.step(dt)
    a, b = o1.get_state(), o2.get_state()
    assert not b[1].any() and np.array_equal(b, np.broadcast_to(b[:, :, :, :1], b.shape))
    for v1, v2 in ((0, 0), (1, 2), (4, 4)):
        assert np.abs(b[v2, 0, :, 0] - a[v1, 0, 0]).max() <= 2e-14 * np.abs(a[v1]).max()


def test_relabelling_unequal_axes_changes_results_only_at_roundoff():
    n, d = (6, 9, 5), (0.1, 0.04, 0.25)
    U = inputs.random_state(*n, seed=12, vamp=0.4)
    o = make(n, 3, d, (PER,) * 6)
    o.set_state(U)
    perm = (2, 0, 1)                                                    # new axis a = old axis perm[a]
    n2 = tuple(n[perm[a]] for a in range(3))
    d2 = tuple(d[perm[a]] for a in range(3))
    o2 = make(n2, 3, d2, (PER,) * 6)
    o2.set_state(inputs.permute_axes(U, perm))
    for _ in range(4):
        dt = o.cfl_dt()
        assert o2.cfl_dt() == dt                                        # a max and a min: order-free
        o.step(dt); o2.step(dt)
    a, b = inputs.permute_axes(o.get_state(), perm), o2.get_state()
    assert np.abs(a - b).max() <= 1e-13 * np.abs(b).max()
