"""Drivers of the z-slab domain decomposition (include/hydro.h, "domain decomposition into z-slabs").

The paper runs the RiemannProblem decomposed over MPI ranks, one GPU each, with a two-layer ghost
exchange after every Runge-Kutta substep and a reduction of the time step every step
 -- through the host; device-to-device exchange is its
stated future work.  Here the exchange stays on the devices.  Every step of the
arithmetic runs in the CUDA library; this module only orders launches, copies and collectives:

  per step:   [smax all-reduced (MAX) -> dt = (cfl/3) dx / smax]
              substep 1 on the interface planes -> exchange of U1's boundary planes
              substep 1 on the interior (overlaps the exchange)
              substep 2 on the interface planes (after the neighbours' planes arrived) -> exchange
              substep 2 on the interior, local max signal speed fused into it

`SlabGroup`  all slabs in ONE process (one GPU, or several GPUs with peer access): the exchange is
             hydro_halo_push, direct stores into the neighbour's ghost planes (NVLink between GPUs),
             ordered by CUDA events; the max is formed on the device.
`SlabRank`   one slab per process under torch.distributed: hydro_halo_pack -> send/recv (NCCL moves
             the packed device buffers over NVLink; gloo, for tests, stages them through the host)
             -> hydro_halo_unpack, and all_reduce(MAX) of the signal speed.
Results are bit-identical to the single-domain run: the same cells see the same ghost values and the
same dt (a maximum is exact in any order).
"""
import numpy as np


def partition(nz, nranks):
    """Planes [k0, k0 + n) of every slab: dealt out evenly, the first nz % nranks get one more
    (the rule of hydro_create_slab)."""
    base, extra = divmod(nz, nranks)
    out, k0 = [], 0
    for r in range(nranks):
        n = base + (1 if r < extra else 0)
        out.append((k0, n))
        k0 += n
    return out


def neighbours(rank, nranks, periodic_z):
    """(low neighbour, high neighbour) of a slab, None at a physical boundary."""
    if nranks == 1:
        return None, None
    lo = rank - 1 if rank > 0 else (nranks - 1 if periodic_z else None)
    hi = rank + 1 if rank < nranks - 1 else (0 if periodic_z else None)
    return lo, hi


class _DevPtr:
    """A raw device pointer as a CUDA-array-interface object (torch.as_tensor wraps it, no copy)."""

    def __init__(self, ptr, n):
        self.__cuda_array_interface__ = {"shape": (n,), "typestr": "<f8", "data": (int(ptr), False),
                                         "version": 2, "strides": None}


class SlabGroup:
    """All slabs of the domain in one process.  `devices`: CUDA device index per slab (default: all
    on the current device).  Same call names as binding.Hydro for the whole-domain operations."""

    def __init__(self, nx, ny, nz, gamma, dx, bc, nslabs, devices=None, verify=False, cfl=0.7,
                 theta=None, variant=None):
        import torch
        from .binding import Hydro, BC_PERIODIC
        self.torch = torch
        self.n = nslabs
        self.shape = (5, nz, ny, nx)
        self.dx, self.cfl = dx, cfl
        self.devices = list(devices) if devices is not None else [torch.cuda.current_device()] * nslabs
        self.parts = partition(nz, nslabs)
        self.nb = [neighbours(r, nslabs, bc[4] == BC_PERIODIC) for r in range(nslabs)]
        self.h = []
        for r in range(nslabs):
            with torch.cuda.device(self.devices[r]):
                h = Hydro(nx, ny, nz, gamma, dx, bc, verify=verify, slab=(r, nslabs))
                h.set_cfl(cfl)
                if theta is not None:
                    h.set_limiter_theta(theta)
                if variant is not None:
                    h.set_kernel_variant(variant)
                self.h.append(h)
        for a in range(nslabs):                            # peer access for direct halo stores
            for b in range(nslabs):
                da, db = self.devices[a], self.devices[b]
                if da != db and not torch.cuda.can_device_access_peer(da, db):
                    raise RuntimeError(f"devices {da} and {db} cannot access each other's memory")
        self.base = [[h.state_base(w) for w in (0, 1)] for h in self.h]
        ev = lambda d: self._on(d, lambda: torch.cuda.Event())      # noqa: E731
        # pushed[w][r]: slab r's boundary planes of buffer w are in its neighbours' ghost planes;
        # done[r]: slab r has finished the step (its stage-2 reads of the second buffer are over)
        self.pushed = [[ev(self.devices[r]) for r in range(nslabs)] for _ in (0, 1)]
        self.done = [ev(self.devices[r]) for r in range(nslabs)]
        self.smax = [self._on(self.devices[r], lambda r=r: torch.as_tensor(_DevPtr(self.h[r].smax_device(), 1),
                                                                           device=f"cuda:{self.devices[r]}"))
                     for r in range(nslabs)]
        self._first = True

    def _on(self, dev, fn):
        with self.torch.cuda.device(dev):
            return fn()

    def close(self):
        for h in self.h:
            h.close()

    # ---- whole-domain state ----
    def set_state(self, U):
        assert tuple(U.shape) == self.shape
        for r, (k0, n) in enumerate(self.parts):
            with self.torch.cuda.device(self.devices[r]):
                self.h[r].set_state(np.ascontiguousarray(U[:, k0:k0 + n]))
        self._first = True

    def get_state(self):
        out = np.empty(self.shape)
        for r, (k0, n) in enumerate(self.parts):
            with self.torch.cuda.device(self.devices[r]):
                out[:, k0:k0 + n] = self.h[r].get_state()
        return out

    def max_signal_speed(self):
        return max(self._on(self.devices[r], self.h[r].max_signal_speed) for r in range(self.n))

    def cfl_dt(self):
        c3 = self.cfl / 3.0
        dxs = self.dx / self.max_signal_speed()
        return c3 * dxs

    def get_time(self):
        return self._on(self.devices[0], self.h[0].get_time)

    # ---- one RK2 step ----
    def _exchange(self, r, which):
        """Slab r pushes its boundary planes of buffer `which` into its neighbours' ghost planes."""
        lo, hi = self.nb[r]
        h = self.h[r]
        for side, peer in ((0, lo), (1, hi)):
            if peer is not None:
                base, pnz, psv = self.base[peer][which]
                h.halo_push(which, side, base, pnz, psv)
        self.pushed[which][r].record(h.torch_stream)

    def _wait_neighbours(self, r, events):
        for peer in self.nb[r]:
            if peer is not None:
                self.h[r].torch_stream.wait_event(events[peer])

    def _step(self, dt):
        """dt > 0: host-supplied; dt == 0: device-resident (smax already all-reduced)."""
        T = self.torch
        for stage, which in ((1, 1), (2, 0)):              # stage 1 writes buffer 1, stage 2 buffer 0
            for r in range(self.n):
                with T.cuda.device(self.devices[r]):
                    if stage == 1:
                        # the neighbours' ghost planes of buffer 1 may be overwritten only after they
                        # finished the previous step; my own ghost planes of buffer 0 must have arrived
                        if not self._first:
                            self._wait_neighbours(r, self.done)
                            self._wait_neighbours(r, self.pushed[0])
                    else:
                        self._wait_neighbours(r, self.pushed[1])
                    self.h[r].substep(stage, dt, 1)
                    self._exchange(r, which)
            for r in range(self.n):
                with T.cuda.device(self.devices[r]):
                    self.h[r].substep(stage, dt, 2)
                    if stage == 2:
                        self.done[r].record(self.h[r].torch_stream)
        self._first = False

    def _initial_exchange(self):
        for r in range(self.n):
            with self.torch.cuda.device(self.devices[r]):
                self._exchange(r, 0)
        for r in range(self.n):
            with self.torch.cuda.device(self.devices[r]):
                self._wait_neighbours(r, self.pushed[0])

    def step(self, dt):
        if self._first:
            self._initial_exchange()
        self._step(dt)

    def _allreduce_smax(self):
        """max over the slabs of the running maximum, in place, on the devices (stream-ordered)."""
        T = self.torch
        if self.n == 1:
            return
        root, s0 = self.devices[0], self.h[0].torch_stream
        with T.cuda.device(root), T.cuda.stream(s0):
            for r in range(1, self.n):
                s0.wait_event(self.done[r])
            vals = [self.smax[r].to(f"cuda:{root}", non_blocking=True) for r in range(self.n)]
            m = T.stack(vals).max(dim=0).values
            self.smax[0].copy_(m)
            ready = T.cuda.Event()
            ready.record(s0)
        for r in range(1, self.n):
            with T.cuda.device(self.devices[r]), T.cuda.stream(self.h[r].torch_stream):
                self.h[r].torch_stream.wait_event(ready)
                self.smax[r].copy_(m, non_blocking=True)

    def run_steps(self, n):
        """n steps with the time step kept on the devices (no host round trip)."""
        if self._first:
            for r in range(self.n):
                with self.torch.cuda.device(self.devices[r]):
                    self.h[r].reduce_smax()
                    self.done[r].record(self.h[r].torch_stream)
            self._initial_exchange()
        for _ in range(n):
            self._allreduce_smax()
            self._step(0.0)

    def synchronize(self):
        for r in range(self.n):
            with self.torch.cuda.device(self.devices[r]):
                self.h[r].torch_stream.synchronize()


class HydroEngine:
    """What SlabRank needs from a slab: binding.Hydro behind five calls (tests pass a stand-in)."""

    def __init__(self, h):
        import torch
        self.h, self.torch = h, torch
        n = h.halo_count()
        self.buf = {(w, s, d): torch.empty(n, dtype=torch.float64, device="cuda")
                    for w in (0, 1) for s in (0, 1) for d in ("send", "recv")}

    def substep(self, stage, dt, part):
        self.h.substep(stage, dt, part)

    def pack(self, which, side):
        b = self.buf[(which, side, "send")]
        self.h.halo_pack(which, side, b)
        return b

    def recv_buffer(self, which, side):
        return self.buf[(which, side, "recv")]

    def unpack(self, which, side, buf):
        self.h.halo_unpack(which, side, buf)

    def local_smax(self):
        return self.h.max_signal_speed()

    def stream(self):
        return self.h.torch_stream

    def reduce_smax(self):
        self.h.reduce_smax()

    def smax_tensor(self):
        """The running maximum of the signal speed on the device, as a 1-element tensor (no copy)."""
        return self.torch.as_tensor(_DevPtr(self.h.smax_device(), 1), device="cuda")


class SlabRank:
    """One slab per process; `dist` is torch.distributed (initialised).  NCCL: the packed device
    buffers go GPU to GPU (NVLink) on a communication stream while the interior planes of the substep
    are computed on the slab's stream; any other backend (gloo, tests): staged through the host."""

    def __init__(self, engine, dist, rank, nranks, periodic_z, dx, cfl=0.7):
        self.e, self.dist, self.rank, self.nranks = engine, dist, rank, nranks
        self.lo, self.hi = neighbours(rank, nranks, periodic_z)
        self.dx, self.cfl = dx, cfl
        self.device_comm = dist.get_backend() == "nccl"
        self._first = True
        self._pending = None
        if self.device_comm:
            import torch
            self.comm_stream = torch.cuda.Stream()

    def _faces(self):
        """(my side, peer) of the interfaces.  A face's planes feed the OTHER side of the peer; both
        ends list their messages by the receiver's side, so two slabs that meet on both faces
        (periodic z, two ranks) still match sends to receives."""
        return [(side, peer) for side, peer in ((0, self.lo), (1, self.hi)) if peer is not None]

    def _start_exchange(self, which):
        """Pack my boundary planes of buffer `which` and start moving them to the neighbours' ghost
        planes (and theirs to mine)."""
        import torch
        dist, faces = self.dist, self._faces()
        if not faces:
            self._pending = (which, [])
            return
        sends = sorted(((1 - side, peer, self.e.pack(which, side)) for side, peer in faces))   # by receiver's side
        recvs = sorted(((side, peer, self.e.recv_buffer(which, side)) for side, peer in faces))
        if self.device_comm:
            packed = torch.cuda.Event()
            packed.record(self.e.stream())
            with torch.cuda.stream(self.comm_stream):
                self.comm_stream.wait_event(packed)
                ops = [dist.P2POp(dist.isend, b, p) for _, p, b in sends] + \
                      [dist.P2POp(dist.irecv, b, p) for _, p, b in recvs]
                for w in dist.batch_isend_irecv(ops):
                    w.wait()
                arrived = torch.cuda.Event()
                arrived.record(self.comm_stream)
            self._pending = (which, [(side, b) for side, _, b in recvs], arrived)
            return
        # host-staged: the copies are ordered on the slab's stream (the library's kernels run there)
        import contextlib
        st = self.e.stream() if hasattr(self.e, "stream") else None
        ctx = torch.cuda.stream(st) if st is not None else contextlib.nullcontext()
        with ctx:
            reqs = [dist.isend(b.cpu(), p, tag=tag) for tag, p, b in sends]      # .cpu() waits for the pack
            host = []
            for side, p, b in recvs:
                hb = torch.empty(b.shape, dtype=b.dtype)
                reqs.append(dist.irecv(hb, p, tag=side))
                host.append((side, b, hb))
            for q in reqs:
                q.wait()
            for side, b, hb in host:
                b.copy_(hb)                       # H2D on the slab's stream, before the unpack
        self._pending = (which, [(side, b) for side, b, _ in host])

    def _finish_exchange(self):
        """The neighbours' planes into my ghost planes (before the substep that reads them)."""
        if self._pending is None:
            return
        which, got = self._pending[0], self._pending[1]
        if self.device_comm and len(self._pending) > 2:
            self.e.stream().wait_event(self._pending[2])
        for side, b in got:
            self.e.unpack(which, side, b)
        self._pending = None

    def cfl_dt(self):
        import torch
        s = torch.tensor([self.e.local_smax()], dtype=torch.float64)
        if self.device_comm:
            s = s.cuda()
        self.dist.all_reduce(s, op=self.dist.ReduceOp.MAX)
        c3 = self.cfl / 3.0
        dxs = self.dx / float(s.item())
        return c3 * dxs

    def run_steps(self, n):
        """n steps with the time step kept on the devices: the running maximum is all-reduced in place
        (NCCL, ordered on the slab's stream) and every slab forms the same dt from it at the start of
        substep 1.  Other backends fall back to the host-side reduction."""
        if not self.device_comm:
            for _ in range(n):
                self.step(self.cfl_dt())
            return
        import torch
        if self._first:
            self.e.reduce_smax()
        smax = self.e.smax_tensor()
        for _ in range(n):
            with torch.cuda.stream(self.e.stream()):
                self.dist.all_reduce(smax, op=self.dist.ReduceOp.MAX)
            self.step(0.0)

    def step(self, dt):
        """dt > 0: host-supplied step; dt == 0: device-resident (run_steps)."""
        if self._first:
            self._start_exchange(0)
            self._first = False
        self._finish_exchange()                  # ghost planes of the state (previous step / initial)
        self.e.substep(1, dt, 1)
        self._start_exchange(1)
        self.e.substep(1, dt, 2)                 # interior: overlaps the transfer
        self._finish_exchange()
        self.e.substep(2, dt, 1)
        self._start_exchange(0)
        self.e.substep(2, dt, 2)
