"""GPU-vs-oracle parity of the 1D / 2D runs and of non-cubic cells (hydro_create_nd; SURVEY.md
section 8(f) NEXT-3, R21-R24).  Verification build: bit-identical to the
oracle (state, time step, clock); production build: the one-step / end-of-run bars of
test_gpu_parity.py."""
import numpy as np
import pytest

from paper_1812_07977_b200 import inputs
from test_gpu_parity import assert_one_step_bar, assert_production_bar

pytestmark = pytest.mark.gpu

OUT, REF, PER = 0, 1, 2


def _pair(shape, ndim, dxyz, bc, gamma=1.4, cfl=0.7, theta=None, verify=True, variant=None):
    from oracle import OracleHydro
    from paper_1812_07977_b200.binding import Hydro
    nx, ny, nz = shape
    g = Hydro(nx, ny, nz, gamma, dxyz[0], bc, verify=verify, ndim=ndim, dxyz=dxyz)
    c = OracleHydro(nx, ny, nz, gamma, dxyz[0], bc, ndim=ndim, dxyz=dxyz)
    for h in (g, c):
        h.set_cfl(cfl)
        if theta is not None:
            h.set_limiter_theta(theta)
    if variant is not None:
        g.set_kernel_variant(variant)
    return g, c


CASES = [
    (1, (257, 1, 1), (0.01, 1.0, 1.0), (OUT, OUT, OUT, OUT, OUT, OUT)),
    (1, (64, 1, 1), (0.3, 1.0, 1.0), (REF, OUT, OUT, OUT, OUT, OUT)),
    (1, (200001, 1, 1), (1e-5, 1.0, 1.0), (OUT, REF, OUT, OUT, OUT, OUT)),    # fused 1D kernel: more tiles than resident blocks
    (1, (1000, 1, 1), (1e-3, 1.0, 1.0), (PER, PER, OUT, OUT, OUT, OUT)),       # periodic x: wrapped source cells
    (1, (2, 1, 1), (0.3, 1.0, 1.0), (PER, PER, OUT, OUT, OUT, OUT)),
    (2, (70, 37, 1), (0.02, 0.02, 1.0), (OUT, REF, PER, PER, OUT, OUT)),
    (2, (33, 5, 1), (0.1, 0.031, 1.0), (PER, PER, REF, OUT, OUT, OUT)),
    (2, (2, 2, 1), (0.1, 0.4, 1.0), (REF, REF, REF, REF, OUT, OUT)),
    (2, (100, 130, 1), (0.01, 0.01, 1.0), (OUT, OUT, OUT, OUT, OUT, OUT)),   # fused 2D kernel: 4 x 9 tiles
    (2, (45, 83, 1), (0.02, 0.013, 1.0), (REF, OUT, OUT, REF, OUT, OUT)),
    (2, (64, 64, 1), (0.02, 0.02, 1.0), (PER, PER, PER, PER, OUT, OUT)),
    (3, (37, 21, 9), (0.1, 0.07, 0.23), (OUT, REF, PER, PER, REF, OUT)),     # fused kernel, non-cubic cells
    (3, (40, 18, 35), (0.05, 0.05, 0.011), (PER, PER, OUT, OUT, REF, REF)),
]


@pytest.mark.parametrize("ndim,shape,dxyz,bc", CASES)
def test_nd_runs_bit_identical_on_verification_build(ndim, shape, dxyz, bc):
    U = inputs.random_state(*shape, seed=sum(shape) + ndim, vamp=0.5)
    variants = {1: (1, 0), 2: (3, 1, 2, 0), 3: (1, 2, 0)}[ndim]
    for variant in variants:
        g, c = _pair(shape, ndim, dxyz, bc, variant=variant)
        if ndim == 2 and variant == 2:
            g.set_tiling(16, 2)                            # several chunks of two tile rows per column
        g.set_state(U); c.set_state(U)
        assert g.get_padded().shape == c.get_padded().shape
        for _ in range(3):
            dt = c.cfl_dt()
            assert g.cfl_dt() == dt
            g.step(dt); c.step(dt)
        assert np.array_equal(g.get_state(), c.get_state()), variant
        g.run_steps(3)                                     # device-resident dt: (cfl/ndim) min(d)/smax
        for _ in range(3):
            c.step(c.cfl_dt())
        assert np.array_equal(g.get_state(), c.get_state()), variant
        assert g.get_time() == c.get_time()
        g.close()


@pytest.mark.parametrize("ndim,shape,dxyz,bc", CASES)
def test_nd_ghost_fill_bit_exact(ndim, shape, dxyz, bc):
    U = inputs.random_state(*shape, seed=5)
    g, c = _pair(shape, ndim, dxyz, bc)
    g.set_state(U); c.set_state(U)
    g.ghost_fill(); c.ghost_fill()
    a, b = g.get_padded(), c.get_padded()
    gh = [np.zeros(n, bool) for n in a.shape[1:]]
    for ax, arr in enumerate(gh):                          # axes z, y, x
        if 2 - ax < ndim:
            arr[:2] = arr[-2:] = True
    nghost = gh[0][:, None, None].astype(int) + gh[1][None, :, None] + gh[2][None, None, :]
    mask = np.broadcast_to(nghost <= 1, a.shape)           # edges / corners are never read
    assert np.array_equal(a[mask], b[mask])


def test_true_1d_sod_evolve_matches_oracle_and_production_bar():
    nx = 512
    U = inputs.sod(nx, 1, 1)
    bc = (OUT,) * 6
    d = (1.0 / nx, 1.0, 1.0)
    g, c = _pair((nx, 1, 1), 1, d, bc)
    g.set_state(U); c.set_state(U)
    ng, nc = g.evolve(0.2), c.evolve(0.2)
    assert ng == nc and g.get_time() == c.get_time() == (0.2, nc)
    assert np.array_equal(g.get_state(), c.get_state())
    gp, _ = _pair((nx, 1, 1), 1, d, bc, verify=False)
    gp.set_state(U)
    assert abs(gp.evolve(0.2) - nc) <= 1
    assert_production_bar(gp.get_state(), c.get_state())


def test_2d_production_build_within_bars():
    n = 96
    a = 2 * np.arange(n, dtype=np.int64) + 1 - n
    inside = 4 * (a[:, None] ** 2 + a[None, :] ** 2) < n * n
    z = np.zeros((1, n, n))
    U = inputs.conserved_from_primitive(np.where(inside, 1.0, 0.125)[None], z, z, z,
                                        np.where(inside, 1.0, 0.1)[None], 1.4)
    g, c = _pair((n, n, 1), 2, (1.0 / n, 1.0 / n, 1.0), (OUT,) * 6, verify=False)
    g.set_state(U); c.set_state(U)
    dt = c.cfl_dt()
    g.step(dt); c.step(dt)
    assert_one_step_bar(g.get_state(), c.get_state(), tol=2e-14)
    g.run_steps(40)
    for _ in range(40):
        c.step(c.cfl_dt())
    assert_production_bar(g.get_state(), c.get_state())


def test_noncubic_3d_production_build_within_bars():
    shape, d = (48, 40, 36), (1.0 / 48, 0.8 / 40, 1.3 / 36)
    U = inputs.random_state(*shape, seed=9, vamp=0.3)
    g, c = _pair(shape, 3, d, (PER,) * 6, gamma=5.0 / 3.0, cfl=0.5, verify=False)
    g.set_state(U); c.set_state(U)
    g.run_steps(10)
    for _ in range(10):
        c.step(c.cfl_dt())
    assert_production_bar(g.get_state(), c.get_state())


def test_create_nd_status_codes():
    from paper_1812_07977_b200.binding import Hydro, HydroError
    for kw in (dict(n=(8, 2, 1), ndim=1), dict(n=(8, 1, 2), ndim=2), dict(n=(1, 1, 1), ndim=1),
               dict(n=(8, 8, 8), ndim=4)):
        with pytest.raises(HydroError) as e:
            Hydro(*kw["n"], 1.4, 0.1, (0,) * 6, ndim=kw["ndim"], dxyz=(0.1, 0.1, 0.1))
        assert e.value.code == 1
    with pytest.raises(HydroError):
        Hydro(8, 8, 1, 1.4, 0.1, (0,) * 6, ndim=2, dxyz=(0.1, -0.1, 0.1))
    g = Hydro(8, 8, 1, 1.4, 0.1, (0,) * 6, ndim=2, dxyz=(0.1, 0.2, 0.1))
    g.set_kernel_variant(3)                                # warp-column kernel: 2D runs only
    g.set_kernel_variant(1); g.set_tiling(16, 4)
    with pytest.raises(HydroError):
        g.set_tiling(8, 4)                                 # 2D runs use 32 x 16 tiles
    g = Hydro(8, 1, 1, 1.4, 0.1, (0,) * 6, ndim=1, dxyz=(0.1, 0.2, 0.1))
    g.set_kernel_variant(0); g.set_kernel_variant(1)       # 1D runs: simple or fused 1D kernel
    with pytest.raises(HydroError):
        g.set_kernel_variant(3)
    with pytest.raises(HydroError):
        g.set_kernel_variant(2)                            # (variant 2 is the 2D / 3D cross-check)
    with pytest.raises(HydroError):
        g.set_tiling(16, 4)


@pytest.mark.gpu
def test_1d_launches_per_step():
    """The fused 1D kernel applies every boundary kind itself (three launches per step: start of step, two
    stages); the simple kernel has its ghost cells filled in memory before each stage (four)."""
    from paper_1812_07977_b200.binding import Hydro
    for bc0, variant, want in ((OUT, 1, 3), (REF, 1, 3), (PER, 1, 3), (OUT, 0, 4)):
        bc = (bc0, bc0, OUT, OUT, OUT, OUT)
        g = Hydro(500, 1, 1, 1.4, 1.0 / 500, bc, ndim=1)
        g.set_kernel_variant(variant)
        g.set_graph_replay(False)
        g.set_state(inputs.random_state(500, 1, 1, seed=5, vamp=0.3))
        g.run_steps(1)
        n0 = g.launch_count()
        g.run_steps(5)
        assert g.launch_count() - n0 == 5 * want, (bc0, variant, g.launch_count() - n0)
        g.close()


@pytest.mark.gpu
def test_2d_variants_agree_bitwise_on_a_large_grid():
    """2D runs of a megacell and more default to the warp-column kernel (variant 3).  On a grid of that
    size -- many strips, many chunks of rows, non-cubic cells, mixed boundaries -- the verification build
    gives the same bits with the warp-column, the tiled and the simple kernel (each of which equals the
    oracle on the small grids above), and the production build stays within the one-step bar of it."""
    import torch
    from paper_1812_07977_b200.binding import Hydro
    nx, ny = 1100, 1000
    bc = (REF, OUT, PER, PER, OUT, OUT)
    U = torch.from_numpy(inputs.random_state(nx, ny, 1, seed=77, vamp=0.4)).cuda()
    out = {}
    for variant in (None, 1, 0):
        g = Hydro(nx, ny, 1, 1.4, 1.0 / nx, bc, verify=True, ndim=2, dxyz=(1.0 / nx, 1.3 / nx, 1.0))
        if variant is not None:
            g.set_kernel_variant(variant)
        g.set_state(U); g.run_steps(3)
        out[variant] = g.get_state()
        g.close()
    assert np.array_equal(out[None], out[1]) and np.array_equal(out[None], out[0])
    g = Hydro(nx, ny, 1, 1.4, 1.0 / nx, bc, verify=False, ndim=2, dxyz=(1.0 / nx, 1.3 / nx, 1.0))
    g.set_state(U); g.run_steps(3)
    assert_one_step_bar(g.get_state(), out[None], tol=6e-14)
    g.close()
