"""Slab decomposition along z.

CPU (`-m "not gpu"`): the partition rule, the neighbour map, and the exchange schedule of
slab.SlabRank on world_size 2 and 3 over gloo, driven with a stand-in engine whose "substep" is an
exact integer stencil: the decomposed run must reproduce the single-domain run of the same stencil,
which it only does when every boundary plane reaches the right ghost plane of the right rank before
the substep that reads it (periodic and open z ends, two slabs meeting on both faces).
GPU: slab.SlabGroup (direct peer stores, one process) and slab.SlabRank (two processes over gloo
sharing the GPU) against the single-domain ORACLE, bit for bit on the verification build."""
import os
import subprocess
import sys
import textwrap

import numpy as np
import pytest

from paper_1812_07977_b200 import inputs, slab

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
OUT, REF, PER = 0, 1, 2


def test_partition_and_neighbours():
    assert slab.partition(10, 3) == [(0, 4), (4, 3), (7, 3)]
    assert slab.partition(8, 4) == [(0, 2), (2, 2), (4, 2), (6, 2)]
    assert slab.partition(7, 1) == [(0, 7)]
    for nz, n in ((256, 8), (37, 5), (11, 3)):
        p = slab.partition(nz, n)
        assert p[0][0] == 0 and sum(c for _, c in p) == nz
        assert all(p[i][0] + p[i][1] == p[i + 1][0] for i in range(n - 1))
        assert max(c for _, c in p) - min(c for _, c in p) <= 1
    assert slab.neighbours(0, 1, True) == (None, None)
    assert slab.neighbours(0, 3, False) == (None, 1) and slab.neighbours(2, 3, False) == (1, None)
    assert slab.neighbours(0, 3, True) == (2, 1) and slab.neighbours(2, 3, True) == (1, 0)
    assert slab.neighbours(0, 2, True) == (1, 1) and slab.neighbours(1, 2, True) == (0, 0)


_FAKE = '''
import os, sys
sys.path.insert(0, {root!r})
import numpy as np, torch, torch.distributed as dist
from paper_1812_07977_b200 import slab

class Engine:
    """Two int64 buffers of planes with 2 ghost planes per side; a substep replaces every active plane
    by an exact integer combination of the 5-plane stencil of the input buffer (stage 2 also of the
    plane's own old value), so any missing, late or misrouted ghost plane changes the result."""
    def __init__(self, planes, zlo_open, zhi_open):
        self.n = len(planes)
        self.buf = [np.zeros(self.n + 4, np.int64), np.zeros(self.n + 4, np.int64)]
        self.buf[0][2:-2] = planes
        self.open = (zlo_open, zhi_open)
    def _fill_open(self, b):
        if self.open[0]: b[0] = b[1] = b[2]
        if self.open[1]: b[-1] = b[-2] = b[-3]
    def substep(self, stage, dt, part):
        if part == 2: return                     # the stand-in does all its planes in part 1
        src, dst = (self.buf[0], self.buf[1]) if stage == 1 else (self.buf[1], self.buf[0])
        self._fill_open(src)
        new = np.array([3 * src[k - 2] + 5 * src[k - 1] + 7 * src[k] + 11 * src[k + 1] + 13 * src[k + 2]
                        for k in range(2, self.n + 2)], np.int64) % 1000003
        if stage == 2: new = (new + dst[2:-2]) % 1000003
        dst[2:-2] = new
    def pack(self, which, side):
        b = self.buf[which]
        return torch.from_numpy((b[2:4] if side == 0 else b[-4:-2]).copy())
    def recv_buffer(self, which, side): return torch.zeros(2, dtype=torch.int64)
    def unpack(self, which, side, t):
        b = self.buf[which]
        if side == 0: b[0:2] = t.numpy()
        else: b[-2:] = t.numpy()
    def local_smax(self): return float(self.buf[0][2:-2].max())

dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
for nz, periodic in ((4 * world + 3, False), (4 * world + 1, True), (2 * world, True)):
    glob = (np.arange(nz, dtype=np.int64) * 7919 + 13) % 1000003
    ref = Engine(glob, not periodic, not periodic)
    if periodic:                                  # single domain: wrap by hand
        class P(Engine):
            def _fill_open(self, b): b[0:2] = b[-4:-2]; b[-2:] = b[2:4]
        ref = P(glob, False, False)
    for _ in range(3):
        ref.substep(1, 1.0, 1); ref.substep(2, 1.0, 1)
    k0, n = slab.partition(nz, world)[rank]
    lo, hi = slab.neighbours(rank, world, periodic)
    e = Engine(glob[k0:k0 + n], lo is None, hi is None)
    drv = slab.SlabRank(e, dist, rank, world, periodic, dx=1.0)
    s = drv.cfl_dt()
    assert s == (0.7 / 3.0) * (1.0 / float(glob.max())), s          # all_reduce(MAX) of the speeds
    for _ in range(3):
        drv.step(1.0)
    assert np.array_equal(e.buf[0][2:-2], ref.buf[0][2 + k0:2 + k0 + n]), (rank, nz, periodic)
print(f"rank{{rank}} ok", flush=True)
dist.destroy_process_group()
'''


def _torchrun(script, nproc, port, env=None, timeout=600):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(nproc),
           "--master-addr", "127.0.0.1", "--master-port", str(port), str(script)]
    e = dict(os.environ, OMP_NUM_THREADS="2")
    e.update(env or {})
    return subprocess.run(cmd, cwd=ROOT, env=e, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True,
                          timeout=timeout)


@pytest.mark.parametrize("world,port", [(2, 29621), (3, 29622)])
def test_slab_rank_exchange_schedule_over_gloo(tmp_path, world, port):
    script = tmp_path / "fake_slab.py"
    script.write_text(_FAKE.format(root=ROOT))
    out = _torchrun(script, world, port)
    assert out.returncode == 0, out.stderr[-3000:]
    for r in range(world):
        assert f"rank{r} ok" in out.stdout


# ---------------------------------------------------------------- GPU: bit-identity with the oracle

def _oracle(shape, gamma, dx, bc, cfl, theta, U, steps):
    from oracle import OracleHydro
    c = OracleHydro(*shape, gamma, dx, bc)
    c.set_cfl(cfl)
    c.set_limiter_theta(theta)
    c.set_state(U)
    for _ in range(steps):
        c.step(c.cfl_dt())
    return c


SLAB_CASES = [
    ((32, 32, 32), (OUT,) * 6, 2, "sphere"),                 # config 0's shape
    ((32, 32, 32), (OUT,) * 6, 3, "sphere"),
    ((37, 21, 23), (OUT, REF, PER, PER, REF, OUT), 3, "random"),        # ragged split 8, 8, 7
    ((40, 12, 9), (PER, PER, OUT, OUT, PER, PER), 2, "random"),         # two slabs meeting on both faces
    ((24, 40, 50), (REF, REF, REF, REF, PER, PER), 4, "random"),
    ((20, 18, 8), (OUT,) * 6, 4, "random"),                  # two planes per slab
]


@pytest.mark.gpu
@pytest.mark.parametrize("shape,bc,nslabs,kind", SLAB_CASES)
def test_slab_group_bit_identical_to_single_domain_oracle(shape, bc, nslabs, kind):
    nx, ny, nz = shape
    U = inputs.sphere(nx) if kind == "sphere" else inputs.random_state(nx, ny, nz, seed=nz + nslabs, vamp=0.5)
    gamma, dx, cfl, theta = 1.4, 1.0 / nx, 0.7, 1.4
    c = _oracle(shape, gamma, dx, bc, cfl, theta, U, 4)
    want, tc = c.get_state(), c.get_time()
    for variant in (1, 2, 0):
        g = slab.SlabGroup(nx, ny, nz, gamma, dx, bc, nslabs, verify=True, cfl=cfl, theta=theta, variant=variant)
        g.set_state(U)
        for _ in range(4):                                 # host-side dt from the max over the slabs
            g.step(g.cfl_dt())
        assert np.array_equal(g.get_state(), want), variant
        g.close()
        g = slab.SlabGroup(nx, ny, nz, gamma, dx, bc, nslabs, verify=True, cfl=cfl, theta=theta, variant=variant)
        g.set_state(U)
        g.run_steps(4)                                     # device-resident dt, max formed on the device
        assert np.array_equal(g.get_state(), want), variant
        assert g.get_time() == tc
        g.close()


@pytest.mark.gpu
def test_slab_group_production_build_config2_shape():
    """128^3 sphere (config 2's shape), 8 slabs of 16 planes, production build, 20 steps."""
    n = 128
    U = inputs.sphere(n)
    c = _oracle((n, n, n), 1.4, 1.0 / n, (OUT,) * 6, 0.7, 1.4, U, 20)
    g = slab.SlabGroup(n, n, n, 1.4, 1.0 / n, (OUT,) * 6, 8)
    g.set_state(U)
    g.run_steps(20)
    from test_gpu_parity import assert_production_bar
    assert_production_bar(g.get_state(), c.get_state())


_RANKS = '''
import os, sys
sys.path.insert(0, {root!r})
sys.path.insert(0, os.path.join({root!r}, "tests"))
import numpy as np, torch, torch.distributed as dist
from paper_1812_07977_b200 import inputs, slab
from paper_1812_07977_b200.binding import Hydro
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
torch.cuda.set_device(0)
for shape, bc in (((32, 32, 32), (0,) * 6), ((37, 21, 23), (0, 1, 2, 2, 2, 2))):
    nx, ny, nz = shape
    U = inputs.sphere(nx) if bc == (0,) * 6 else inputs.random_state(nx, ny, nz, seed=4, vamp=0.5)
    h = Hydro(nx, ny, nz, 1.4, 1.0 / nx, bc, verify=True, slab=(rank, world))
    k0, n = slab.partition(nz, world)[rank]
    assert (h.k_first, h.shape[1]) == (k0, n)
    h.set_state(np.ascontiguousarray(U[:, k0:k0 + n]))
    drv = slab.SlabRank(slab.HydroEngine(h), dist, rank, world, bc[4] == 2, 1.0 / nx)
    for _ in range(4):
        drv.step(drv.cfl_dt())
    got = h.get_state()
    if rank == 0:
        import oracle
        c = oracle.OracleHydro(nx, ny, nz, 1.4, 1.0 / nx, bc)
        c.set_state(U)
        for _ in range(4):
            c.step(c.cfl_dt())
        want = torch.from_numpy(c.get_state())
    else:
        want = torch.empty((5, nz, ny, nx), dtype=torch.float64)
    dist.broadcast(want, 0)
    assert np.array_equal(got, want.numpy()[:, k0:k0 + n]), (rank, shape)
print(f"rank{{rank}} ok", flush=True)
dist.destroy_process_group()
'''


@pytest.mark.gpu
def test_slab_ranks_two_processes_over_gloo_bit_identical(tmp_path):
    script = tmp_path / "ranks.py"
    script.write_text(_RANKS.format(root=ROOT))
    out = _torchrun(script, 2, 29623)
    assert out.returncode == 0, (out.stdout[-1500:], out.stderr[-3000:])
    assert "rank0 ok" in out.stdout and "rank1 ok" in out.stdout


@pytest.mark.gpu
def test_bench_slab_mode_two_ranks_share_one_gpu_over_gloo():
    """bench.py --decomp slab end to end: two slab ranks of one 32 x 32 x 64 domain (they share the
    GPU and meet only on the host), one JSON line from rank 0."""
    import json
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", "29624", "bench.py", "--gpus", "2", "--decomp", "slab",
           "--config", "0", "--steps", "10", "--warmup", "3"]
    env = dict(os.environ, HYDRO_BENCH_BACKEND="gloo", OMP_NUM_THREADS="2")
    out = subprocess.run(cmd, cwd=ROOT, env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True, timeout=600)
    assert out.returncode == 0, out.stderr[-3000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["n_gpus"] == 2 and d["value"] > 0 and d["devices_shared"] and "z-slabs" in d["config"]["parallelism"]
    assert d["gpu_launches"] >= 10 * 5
