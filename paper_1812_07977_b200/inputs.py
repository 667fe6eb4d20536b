"""Seeded synthetic inputs for BASELINE.json's configs (recipe R10).

This module serves both the CUDA path and the oracle and holds none of the method's
arithmetic: it only writes initial conserved states ``U[5][nz][ny][nx]`` (x fastest, active
cells only, fp64) from primitive data, ``E = p/(gamma-1) + rho |v|^2 / 2``.
It imports neither side.
"""
from dataclasses import dataclass, field

import numpy as np

BC_OUTFLOW, BC_REFLECT, BC_PERIODIC = 0, 1, 2


def conserved_from_primitive(rho, vx, vy, vz, p, gamma):
    """Pack primitive fields (arrays of equal shape [nz,ny,nx]) into U[5,nz,ny,nx]."""
    rho = np.asarray(rho, dtype=np.float64)
    U = np.empty((5,) + rho.shape, dtype=np.float64)
    U[0] = rho
    U[1] = rho * vx
    U[2] = rho * vy
    U[3] = rho * vz
    U[4] = p / (gamma - 1.0) + 0.5 * rho * (vx * vx + vy * vy + vz * vz)
    return U


def sphere(n, gamma=1.4, rho_in=1.0, p_in=1.0, rho_out=0.125, p_out=0.1):
    """Spherical Riemann problem on [0,1]^3 with n^3 cells (configs 0, 2, 3).

    A cell is inside iff its centre lies within radius 0.25 of (1/2,1/2,1/2); evaluated in
    integers (a=2i+1-n etc., inside iff a^2+b^2+c^2 < n^2/4) so that no rounding decides it.
    """
    a = 2 * np.arange(n, dtype=np.int64) + 1 - n
    r2 = a[:, None, None] ** 2 + a[None, :, None] ** 2 + a[None, None, :] ** 2
    inside = 4 * r2 < n * n
    rho = np.where(inside, rho_in, rho_out)
    p = np.where(inside, p_in, p_out)
    z = np.zeros_like(rho)
    return conserved_from_primitive(rho, z, z, z, p, gamma)


def sod(nx, ny=4, nz=4, gamma=1.4):
    """1D Sod tube along x embedded in 3D (config 1): left state (1, 0, 1) for cell centres
    x < 0.5, right state (0.125, 0, 0.1).  Centres never equal 0.5 for even `nx`."""
    left = (2 * np.arange(nx) + 1) < nx
    left3 = np.broadcast_to(left[None, None, :], (nz, ny, nx))
    rho = np.where(left3, 1.0, 0.125)
    p = np.where(left3, 1.0, 0.1)
    z = np.zeros((nz, ny, nx))
    return conserved_from_primitive(rho, z, z, z, p, gamma)


def permute_axes(U, perm):
    """Relabel axes of a packed state: new axis a is old axis perm[a] (0=x,1=y,2=z).
    Returns the state of the relabelled problem (momenta permuted accordingly)."""
    # numpy axis of spatial axis a in U[v, z, y, x] is 3 - a
    out = np.transpose(U, (0,) + tuple(3 - perm[2 - k] for k in range(3)))
    out = out[[0, 1 + perm[0], 1 + perm[1], 1 + perm[2], 4]]
    return np.ascontiguousarray(out)


def reflect_axis(U, a):
    """Mirror a packed state along spatial axis a (normal momentum changes sign)."""
    out = np.flip(U, axis=3 - a).copy()
    out[1 + a] = -out[1 + a]
    return out


def noise(nx, ny=None, nz=None, gamma=5.0 / 3.0, seed=12345, amp=0.1):
    """Config 4: rho=1+amp*u0, p=1+amp*u1, v_e=amp*u_{2+e}, u iid Uniform(-1,1) per cell."""
    ny = nx if ny is None else ny
    nz = nx if nz is None else nz
    rng = np.random.default_rng(seed)
    u = rng.uniform(-1.0, 1.0, (5, nz, ny, nx))
    return conserved_from_primitive(1.0 + amp * u[0], amp * u[2], amp * u[3], amp * u[4],
                                    1.0 + amp * u[1], gamma)


def random_state(nx, ny, nz, gamma=1.4, seed=0, vamp=0.5):
    """Positive random state for unit tests: rho,p in (0.5,1.5), |v_e| < vamp."""
    rng = np.random.default_rng(seed)
    u = rng.uniform(-1.0, 1.0, (5, nz, ny, nx))
    return conserved_from_primitive(1.0 + 0.5 * u[0], vamp * u[2], vamp * u[3], vamp * u[4],
                                    1.0 + 0.5 * u[1], gamma)


@dataclass
class Config:
    """One row of BASELINE.json:configs."""
    name: str
    shape: tuple                 # (nx, ny, nz)
    gamma: float
    cfl: float
    bc: tuple                    # xlo,xhi,ylo,yhi,zlo,zhi
    dx: float
    steps: int = 0               # number of {cfl_dt, step} pairs; 0 -> use t_final
    t_final: float = 0.0
    theta: float = 1.4
    make: object = field(default=None, repr=False)
    index: int = -1

    @property
    def cells(self):
        return self.shape[0] * self.shape[1] * self.shape[2]

    def state(self):
        return self.make()


_OUT6 = (BC_OUTFLOW,) * 6
_PER6 = (BC_PERIODIC,) * 6


def config(i):
    """BASELINE.json:configs[i] as a Config."""
    if i == 0:
        return Config("cfg0_sphere32", (32, 32, 32), 1.4, 0.7, _OUT6, 1.0 / 32, steps=20,
                      make=lambda: sphere(32))
    if i == 1:
        return Config("cfg1_sod512x4x4", (512, 4, 4), 1.4, 0.7,
                      (BC_OUTFLOW, BC_OUTFLOW, BC_PERIODIC, BC_PERIODIC, BC_PERIODIC, BC_PERIODIC),
                      1.0 / 512, t_final=0.2, make=lambda: sod(512, 4, 4))
    if i == 2:
        return Config("cfg2_sphere128", (128, 128, 128), 1.4, 0.7, _OUT6, 1.0 / 128, steps=100,
                      make=lambda: sphere(128))
    if i == 3:
        return Config("cfg3_sphere256", (256, 256, 256), 1.4, 0.7, _OUT6, 1.0 / 256, steps=200,
                      make=lambda: sphere(256))
    if i == 4:
        return Config("cfg4_noise512", (512, 512, 512), 5.0 / 3.0, 0.5, _PER6, 1.0 / 512,
                      steps=50, make=lambda: noise(512))
    raise ValueError(i)


_config_raw = config


def config(i):  # noqa: F811
    """BASELINE.json:configs[i] as a Config (with .index set)."""
    c = _config_raw(i)
    c.index = i
    return c
