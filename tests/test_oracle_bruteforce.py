"""P5: one RK2 step of single cells written out in scalar Python (IEEE doubles, no FMA) from
DESIGN.md's O1-O6, with the ghost rule expressed as an index map instead of a fill.  Pins the
oracle's indexing, ghost use, loop bounds and RK wiring on tiny grids with every boundary type on
every face.  Shares no code with the oracle or the CUDA path."""
import math

import numpy as np
import pytest

from oracle import OracleHydro
from paper_1812_07977_b200 import inputs

OUT, REF, PER = 0, 1, 2
THETA = 1.4


def s3(a, b, c):
    x = sorted((a, b, c))
    return (x[0] + x[2]) + x[1]


def prim(U, g):
    inv = 1.0 / U[0]
    vx, vy, vz = U[1] * inv, U[2] * inv, U[3] * inv
    q = s3(vx * vx, vy * vy, vz * vz)
    return (U[0], vx, vy, vz, (g - 1.0) * (U[4] - (0.5 * U[0]) * q))


def slope(wm, w0, wp):
    a, b = w0 - wm, wp - w0
    m = min(THETA * abs(a), THETA * abs(b), 0.5 * abs(a + b))
    if a > 0 and b > 0:
        return m
    if a < 0 and b < 0:
        return -m
    return 0.0


def side(W, d, g):
    rho, p = W[0], W[4]
    v = W[1:4]
    vn, vt1, vt2 = v[d], v[(d + 1) % 3], v[(d + 2) % 3]
    c = math.sqrt((g * p) / rho)
    k = vn * vn + (vt1 * vt1 + vt2 * vt2)
    E = p * (1.0 / (g - 1.0)) + (0.5 * rho) * k
    U = [rho, rho * v[0], rho * v[1], rho * v[2], E]
    F = [U[1 + d], U[1] * vn, U[2] * vn, U[3] * vn, (E + p) * vn]
    F[1 + d] = F[1 + d] + p
    return U, F, vn, c


def hll(WL, WR, d, g):
    UL, FL, vL, cL = side(WL, d, g)
    UR, FR, vR, cR = side(WR, d, g)
    ap = max(0.0, vL + cL, vR + cR)
    am = max(0.0, cL - vL, cR - vR)
    w = 1.0 / (ap + am)
    pi = ap * am
    return [((ap * FL[v] + am * FR[v]) - pi * (UR[v] - UL[v])) * w for v in range(5)]


class Grid:
    """Conserved state on active cells + boundary rule as an index map (R9)."""

    def __init__(self, get_active, n, bc):
        self.get_active, self.n, self.bc = get_active, n, bc

    def U(self, idx):
        """Conserved state at 0-based active index idx (each component may be -2..n+1)."""
        idx = list(idx)
        sign = [1.0] * 5
        for a in range(3):
            n, i = self.n[a], idx[a]
            if i < 0:
                kind = self.bc[2 * a]
                if kind == OUT:
                    i = 0
                elif kind == PER:
                    i = i + n
                else:
                    i = -1 - i
                    sign[1 + a] = -sign[1 + a]
            elif i >= n:
                kind = self.bc[2 * a + 1]
                if kind == OUT:
                    i = n - 1
                elif kind == PER:
                    i = i - n
                else:
                    i = 2 * n - 1 - i
                    sign[1 + a] = -sign[1 + a]
            idx[a] = i
        u = self.get_active(tuple(idx))
        return tuple(s * x for s, x in zip(sign, u))


def delta_U(grid, idx, g, r):
    """-(dt/dx) * sum3 of the three flux differences at active cell idx (O2-O5)."""
    dF = []
    for d in range(3):
        def W(o):
            j = list(idx)
            j[d] += o
            return prim(grid.U(j), g)
        Wm2, Wm1, W0, Wp1, Wp2 = W(-2), W(-1), W(0), W(1), W(2)
        sm1 = [slope(Wm2[v], Wm1[v], W0[v]) for v in range(5)]
        s0 = [slope(Wm1[v], W0[v], Wp1[v]) for v in range(5)]
        sp1 = [slope(W0[v], Wp1[v], Wp2[v]) for v in range(5)]
        outer_m1 = [Wm1[v] + 0.5 * sm1[v] for v in range(5)]
        inner_0 = [W0[v] - 0.5 * s0[v] for v in range(5)]
        outer_0 = [W0[v] + 0.5 * s0[v] for v in range(5)]
        inner_p1 = [Wp1[v] - 0.5 * sp1[v] for v in range(5)]
        Fm = hll(outer_m1, inner_0, d, g)
        Fp = hll(outer_0, inner_p1, d, g)
        dF.append([Fp[v] - Fm[v] for v in range(5)])
    return [-(r * s3(dF[0][v], dF[1][v], dF[2][v])) for v in range(5)]


def rk2_cell(U0arr, n, bc, g, dt, dx, idx):
    r = dt / dx
    g0 = Grid(lambda j: tuple(U0arr[:, j[2], j[1], j[0]].tolist()), n, bc)
    memo = {}

    def U1(j):
        if j not in memo:
            u0 = g0.U(j)
            du = delta_U(g0, j, g, r)
            memo[j] = tuple(u0[v] + du[v] for v in range(5))
        return memo[j]

    g1 = Grid(U1, n, bc)
    u0, u1 = g0.U(idx), U1(tuple(idx))
    du = delta_U(g1, idx, g, r)
    return [0.5 * ((u0[v] + u1[v]) + du[v]) for v in range(5)]


CASES = [
    ((OUT,) * 6, (4, 5, 6)),
    ((PER,) * 6, (4, 4, 5)),
    ((REF,) * 6, (5, 4, 4)),
    ((OUT, REF, PER, PER, REF, OUT), (4, 6, 5)),
    ((REF, OUT, REF, REF, PER, PER), (6, 4, 4)),
    ((PER, PER, OUT, REF, OUT, OUT), (2, 3, 2)),     # smallest legal sizes: ghosts wrap twice
]


@pytest.mark.parametrize("bc,n", CASES)
def test_single_cell_rk2_update_matches_hand_expansion_bitwise(bc, n):
    nx, ny, nz = n
    g, dx = 1.4, 0.1
    U0 = inputs.random_state(nx, ny, nz, gamma=g, seed=sum(n) + sum(bc), vamp=0.6)
    o = OracleHydro(nx, ny, nz, g, dx, bc)
    o.set_state(U0)
    dt = o.cfl_dt()
    o.step(dt)
    got = o.get_state()
    cells = {(0, 0, 0), (nx - 1, ny - 1, nz - 1), (0, ny - 1, 0), (nx - 1, 0, nz - 1),
             (nx // 2, ny // 2, nz // 2), (1, 0, nz - 2), (nx - 2, 1, 0)}
    for idx in sorted(cells):
        want = rk2_cell(U0, n, bc, g, dt, dx, idx)
        have = got[:, idx[2], idx[1], idx[0]].tolist()
        assert have == want, (idx, have, want)


def test_time_step_matches_hand_expansion():
    g, dx, cfl = 5.0 / 3.0, 0.05, 0.5
    U0 = inputs.random_state(4, 3, 5, gamma=g, seed=99)
    o = OracleHydro(4, 3, 5, g, dx, (PER,) * 6)
    o.set_cfl(cfl)
    o.set_state(U0)
    smax = 0.0
    for k in range(5):
        for j in range(3):
            for i in range(4):
                U = U0[:, k, j, i].tolist()
                inv = 1.0 / U[0]
                vx, vy, vz = U[1] * inv, U[2] * inv, U[3] * inv
                q = s3(vx * vx, vy * vy, vz * vz)
                p = (g - 1.0) * (U[4] - (0.5 * U[0]) * q)
                smax = max(smax, math.sqrt(q) + math.sqrt((g * p) * inv))
    assert o.max_signal_speed() == smax
    assert o.cfl_dt() == (cfl / 3.0) * (dx / smax)
