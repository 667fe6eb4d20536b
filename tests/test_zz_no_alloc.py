"""hydro_max_signal_speed_noalloc: the allocation-free entry point (include/hydro.h) against the
existing path (a handle's hydro_max_signal_speed), two calls in a row and more.

The entry point keeps the scratch of the reduction in a file-scope device array that every call
shares and that keeps the last call's contents; the cases are ordered so that a call which trusted
stale contents (partials or the ticket of the previous, larger call) would fail.  Collected last
(file name): the suite runs with pytest -x.  Passes alone in a fresh process and after the others.

Bars (those of tests/test_gpu_parity.py): the maximum is the same arithmetic on the same cells in both
paths (cell_signal_speed, O7): bit for bit on the verification build; within the one-step bar, 1e-14
relative, on the production build (separately compiled kernels; after steps the handle's value comes
from the fused stage-2 epilogue's regrouped arithmetic); the flag is exact.
"""
import ctypes as C

import numpy as np
import pytest

from paper_1812_07977_b200 import binding, inputs

OUT6 = (0,) * 6


def _existing(U, gamma, verify):
    """max(|v| + c_s) through the existing path: a handle, hydro_set_state, hydro_max_signal_speed."""
    nz, ny, nx = U.shape[1:]
    h = binding.Hydro(nx, ny, nz, gamma, 1.0 / nx, OUT6, verify=verify)
    h.set_state(U)
    s = h.max_signal_speed()
    h.close()
    return s


def _same(got, want, verify):
    """Bit for bit on the verification build (-fmad=false); on the production build the two kernels are
    compiled separately and may contract differently: the one-step bar, 1e-14 relative."""
    return got == want if verify else abs(got - want) <= 1e-14 * want


@pytest.mark.gpu
@pytest.mark.parametrize("verify", [True, False])
def test_two_calls_in_a_row_match_the_existing_path(verify):
    import torch
    dev = torch.device("cuda:0")
    smax = torch.full((1,), -1.0, dtype=torch.float64, device=dev)
    flag = torch.full((1,), -1, dtype=torch.int32, device=dev)
    # call 1: 96 x 80 x 70 = 537 600 cells = 262.5 blocks (ragged tail), fast flow: large partials
    # call 2: 17 x 5 x 3 = 255 cells = one partly filled block, slow flow: every stale partial of call 1
    #         is larger than the right answer
    # call 3: the first state again (same bits as call 1)
    big = inputs.random_state(96, 80, 70, gamma=1.4, seed=3, vamp=3.0)
    small = inputs.random_state(17, 5, 3, gamma=1.4, seed=4, vamp=0.01)
    want_big = _existing(big, 1.4, verify)
    want_small = _existing(small, 1.4, verify)
    assert want_small < 0.75 * want_big
    got = []
    for U in (big, small, big):
        Ud = torch.from_numpy(U).to(dev)
        binding.max_signal_speed_noalloc(Ud, 1.4, smax, flag, verify=verify)
        torch.cuda.synchronize()
        got.append((smax.item(), flag.item()))
    for (s, f), want in zip(got, (want_big, want_small, want_big)):
        assert f == 0
        assert _same(s, want, verify), (s, want)
    assert got[2] == got[0]


@pytest.mark.gpu
def test_after_steps_and_back_to_back_on_one_stream():
    """Config 0 after 3 RK2 steps: the handle's value is the fused stage-2 reduction; the entry point reads
    the same state from hydro_get_state's device copy.  Then 20 calls back to back on one stream with no
    synchronisation in between, alternating two states: each call's outputs land in their own slots."""
    import torch
    dev = torch.device("cuda:0")
    cfg = inputs.config(0)
    for verify in (True, False):
        h = binding.Hydro(*cfg.shape, cfg.gamma, cfg.dx, cfg.bc, verify=verify)
        h.set_cfl(cfg.cfl)
        h.set_state(cfg.state())
        for _ in range(3):
            h.step(h.cfl_dt())
        want = h.max_signal_speed()
        Ud = torch.empty(h.shape, dtype=torch.float64, device=dev)
        h.get_state(Ud)
        h.close()
        smax = torch.zeros(1, dtype=torch.float64, device=dev)
        flag = torch.zeros(1, dtype=torch.int32, device=dev)
        binding.max_signal_speed_noalloc(Ud, cfg.gamma, smax, flag, verify=verify)
        torch.cuda.synchronize()
        if verify:
            assert smax.item() == want
        assert abs(smax.item() - want) <= 1e-14 * want
        assert flag.item() == 0
    a = torch.from_numpy(inputs.random_state(200, 33, 9, seed=5, vamp=2.0)).to(dev)
    b = torch.from_numpy(inputs.random_state(64, 64, 64, seed=6, vamp=0.2)).to(dev)
    outs = torch.zeros(20, dtype=torch.float64, device=dev)
    flags = torch.full((20,), -1, dtype=torch.int32, device=dev)
    for i in range(20):
        binding.max_signal_speed_noalloc(a if i % 2 == 0 else b, 1.4, outs[i:i + 1], flags[i:i + 1])
    torch.cuda.synchronize()
    o = outs.cpu().numpy()
    assert (o[0::2] == o[0]).all() and (o[1::2] == o[1]).all() and o[0] > 2.0 * o[1]
    assert _same(o[0], _existing(a.cpu().numpy(), 1.4, False), False)
    assert _same(o[1], _existing(b.cpu().numpy(), 1.4, False), False)
    assert (flags.cpu().numpy() == 0).all()


@pytest.mark.gpu
def test_unphysical_flag_and_clean_flag_afterwards():
    """rho <= 0 in the last cell of a ragged tail sets the flag (as HYDRO_ERR_UNPHYSICAL does on the
    handle); the next call on a clean state reports 0 again: the flag is not sticky in the scratch."""
    import torch
    dev = torch.device("cuda:0")
    U = inputs.random_state(50, 41, 3, seed=8)
    bad = U.copy()
    bad[0, -1, -1, -1] = -1.0
    smax = torch.zeros(1, dtype=torch.float64, device=dev)
    flag = torch.zeros(1, dtype=torch.int32, device=dev)
    binding.max_signal_speed_noalloc(torch.from_numpy(bad).to(dev), 1.4, smax, flag)
    torch.cuda.synchronize()
    assert flag.item() == 1
    with pytest.raises(binding.HydroError) as e:
        _existing(bad, 1.4, False)
    assert e.value.code == 4
    binding.max_signal_speed_noalloc(torch.from_numpy(U).to(dev), 1.4, smax, flag)
    torch.cuda.synchronize()
    assert flag.item() == 0 and _same(smax.item(), _existing(U, 1.4, False), False)


@pytest.mark.gpu
def test_allocates_nothing_and_rejects_host_pointers():
    """The device's free memory does not move across 50 calls (the first call, which looks up the scratch
    address, is made before the measurement); a host pointer is refused with HYDRO_ERR_ARG."""
    import torch
    dev = torch.device("cuda:0")
    L = binding.load_library(False)
    Ud = torch.from_numpy(inputs.random_state(128, 128, 64, seed=9)).to(dev)
    smax = torch.zeros(1, dtype=torch.float64, device=dev)
    flag = torch.zeros(1, dtype=torch.int32, device=dev)
    binding.max_signal_speed_noalloc(Ud, 1.4, smax, flag)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info(dev)
    for _ in range(50):
        binding.max_signal_speed_noalloc(Ud, 1.4, smax, flag)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info(dev)
    assert free1 == free0
    host = np.ones((5, 64), dtype=np.float64)
    rc = L.hydro_max_signal_speed_noalloc(C.c_void_p(host.ctypes.data), 64, 1.4, C.c_void_p(smax.data_ptr()),
                                          C.c_void_p(flag.data_ptr()), None)
    assert rc == 1 and b"not a device pointer" in L.hydro_last_error()


@pytest.mark.gpu
def test_captured_into_a_cuda_graph_and_replayed():
    """What the entry point is for: captured into a CUDA graph (torch's capture runs in the mode in which
    a cudaMalloc anywhere in the process invalidates the capture), then replayed on changing inputs.  The
    first call on the device -- the set-up that looks up the scratch address -- is made outside capture."""
    import torch
    dev = torch.device("cuda:0")
    a = inputs.random_state(70, 60, 50, seed=11, vamp=1.0)
    b = inputs.random_state(70, 60, 50, seed=12, vamp=4.0)
    Ud = torch.from_numpy(a).to(dev)
    smax = torch.zeros(1, dtype=torch.float64, device=dev)
    flag = torch.zeros(1, dtype=torch.int32, device=dev)
    binding.max_signal_speed_noalloc(Ud, 1.4, smax, flag)
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        binding.max_signal_speed_noalloc(Ud, 1.4, smax, flag)       # on the capturing stream
    for U in (a, b, a):
        Ud.copy_(torch.from_numpy(U))
        smax.fill_(-1.0)
        flag.fill_(-1)
        graph.replay()
        torch.cuda.synchronize()
        assert flag.item() == 0 and _same(smax.item(), _existing(U, 1.4, False), False)


def test_sizes_beyond_the_scratch_are_rejected_without_a_device():
    """Argument errors come before any CUDA call: a size beyond HYDRO_NOALLOC_MAX_CELLS (the capacity of
    the static scratch array), an empty state, a NULL pointer, gamma <= 1."""
    L = binding.load_library(False)
    p = C.c_void_p(256)                      # never dereferenced: the checks below fail first
    call = L.hydro_max_signal_speed_noalloc
    assert binding.NOALLOC_MAX_CELLS == 512 ** 3
    assert call(p, binding.NOALLOC_MAX_CELLS + 1, 1.4, p, p, None) == 1
    msg = L.hydro_last_error()
    assert b"HYDRO_NOALLOC_MAX_CELLS" in msg and b"134217728" in msg
    assert call(p, 0, 1.4, p, p, None) == 1
    assert call(None, 8, 1.4, p, p, None) == 1
    assert call(p, 8, 1.4, None, p, None) == 1
    assert call(p, 8, 1.4, p, None, None) == 1
    assert call(p, 8, 1.0, p, p, None) == 1
    header = open(binding._build.HERE + "/../include/hydro.h").read()
    assert "#define HYDRO_NOALLOC_MAX_CELLS 134217728LL" in header
