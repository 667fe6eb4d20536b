"""P2: the 1D Sod tube embedded in 3D converges in L1 to the exact Riemann solution
(BASELINE.json:configs[1]; "extension of the classic 1D Sod shock tube")."""
import os

import numpy as np

import exact_riemann as er
import oracle
from oracle import OracleHydro, BC_OUTFLOW, BC_PERIODIC
from paper_1812_07977_b200 import inputs

GOLD = os.path.join(os.path.dirname(__file__), "golden", "sod_star_values.txt")
SOD = (1.0, 0.0, 1.0, 0.125, 0.0, 0.1, 1.4)
BC = (BC_OUTFLOW, BC_OUTFLOW, BC_PERIODIC, BC_PERIODIC, BC_PERIODIC, BC_PERIODIC)


def test_exact_solver_reproduces_textbook_star_values():
    gold = {}
    for line in open(GOLD):
        if line.strip() and not line.startswith("#"):
            k, v = line.split()
            gold[k] = float(v)
    ps, us = er.star_state(*SOD)
    assert abs(ps - gold["p_star"]) < 1e-6 and abs(us - gold["u_star"]) < 1e-6
    rho, u, p = er.sample([0.5, 1.2], *SOD)            # between fan tail and contact; contact..shock
    assert abs(rho[0] - gold["rho_star_L"]) < 1e-6 and abs(rho[1] - gold["rho_star_R"]) < 1e-6
    S = gold["shock_speed"]
    rho, _, _ = er.sample([S - 1e-4, S + 1e-4], *SOD)
    assert abs(rho[0] - gold["rho_star_R"]) < 1e-6 and rho[1] == 0.125


def _l1_errors(nx, t_final=0.2):
    o = OracleHydro(nx, 4, 4, 1.4, 1.0 / nx, BC)
    o.set_state(inputs.sod(nx, 4, 4))
    nsteps = o.evolve(t_final)
    U = o.get_state()
    assert o.get_time()[0] == t_final
    # P2 addendum: rows identical, transverse momenta exactly zero
    assert np.array_equal(U, np.broadcast_to(U[:, :1, :1, :], U.shape))
    assert not U[2].any() and not U[3].any()
    x = (np.arange(nx) + 0.5) / nx
    rho_e, u_e, p_e = er.sample((x - 0.5) / t_final, *SOD)
    rho = U[0, 0, 0]
    u = U[1, 0, 0] / rho
    p = 0.4 * (U[4, 0, 0] - 0.5 * rho * u * u)
    dx = 1.0 / nx
    return (np.abs(rho - rho_e).sum() * dx, np.abs(u - u_e).sum() * dx,
            np.abs(p - p_e).sum() * dx, nsteps)


def test_sod_l1_error_falls_with_resolution():
    nth = oracle.get_threads()
    oracle.set_threads(1)                  # 8192-cell grids: thread fork/join would dominate
    try:
        res = {nx: _l1_errors(nx) for nx in (64, 128, 256, 512)}
    finally:
        oracle.set_threads(nth)
    for a, b in ((64, 128), (128, 256), (256, 512)):
        for q, need in ((0, 1.6), (1, 1.5), (2, 1.6)):    # rho, u, p
            assert res[a][q] / res[b][q] >= need, (a, b, q, res[a][q], res[b][q])
    # absolute level at the config-1 resolution (SURVEY.md P2 probe: L1(rho)=1.31e-3, L1(p)=8.61e-4)
    assert res[512][0] < 1.5e-3 and res[512][2] < 1.0e-3
    assert 900 <= res[512][3] <= 1000               # ~960 steps under reading R8
