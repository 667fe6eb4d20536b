"""Host mirror with selected-field, overlapped transfers (the paper's
StorageForm UpdateDevice / UpdateHost, and pinned host memory)."""
import numpy as np
import pytest

from paper_1812_07977_b200 import inputs

pytestmark = pytest.mark.gpu
OUT, PER = 0, 2


def _h(shape, verify=True, bc=(OUT,) * 6):
    from paper_1812_07977_b200.binding import Hydro
    return Hydro(*shape, 1.4, 1.0 / shape[0], bc, verify=verify)


def test_whole_state_and_selected_fields_round_trip():
    shape = (37, 9, 6)
    U = inputs.random_state(*shape, seed=1)
    V = inputs.random_state(*shape, seed=2)
    g = _h(shape)
    pin = g.host_alloc()
    assert pin.shape == (5, 6, 9, 37)
    pin[...] = U
    g.update_device(pin)                               # all five fields
    assert np.array_equal(g.get_state(), U)
    out = g.host_alloc()
    out[...] = -7.0
    g.update_host(out)
    g.transfer_sync()
    assert np.array_equal(out, U)
    pin[...] = V
    g.update_device(pin, fields=1 | 16)                # rho and E only
    want = U.copy(); want[0] = V[0]; want[4] = V[4]
    assert np.array_equal(g.get_state(), want)
    out[...] = -7.0
    g.update_host(out, fields=2 | 4)                   # m_x, m_y only
    g.transfer_sync()
    assert np.array_equal(out[1:3], want[1:3]) and (out[[0, 3, 4]] == -7.0).all()


def test_update_device_is_set_state_without_touching_the_clock():
    from paper_1812_07977_b200.binding import HydroError
    c = inputs.config(0)
    U = c.state()
    a, b = _h(c.shape), _h(c.shape)
    with pytest.raises(HydroError):
        b.update_device(np.ascontiguousarray(U), fields=3)      # first update must bring everything
    a.set_state(U)
    b.update_device(np.ascontiguousarray(U))
    for h in (a, b):
        h.set_cfl(c.cfl)
    for _ in range(3):
        dt = a.cfl_dt()
        assert b.cfl_dt() == dt
        a.step(dt); b.step(dt)
    assert np.array_equal(a.get_state(), b.get_state())
    t = b.get_time()
    b.update_device(np.ascontiguousarray(U), fields=31)
    assert b.get_time() == t and np.array_equal(b.get_state(), U)
    with pytest.raises(HydroError):
        b.update_host(np.empty(b.shape), fields=0)


def test_pipelined_transfers_overlap_steps_without_mixing_them_up():
    """No host synchronisation between iterations: input k+1 goes up while step k runs and result k
    comes down.  Every result must equal the serial set_state / step / get_state path."""
    shape = (64, 48, 40)
    g, ref = _h(shape, bc=(PER,) * 6), _h(shape, bc=(PER,) * 6)
    ins = [inputs.random_state(*shape, seed=10 + k, vamp=0.3) for k in range(5)]
    pins = [g.host_alloc() for _ in range(5)]
    outs = [g.host_alloc() for _ in range(5)]
    for p, u in zip(pins, ins):
        p[...] = u
    dt = 1e-3
    for k in range(5):
        g.update_device(pins[k])
        g.step(dt)
        g.update_host(outs[k])
    g.transfer_sync()
    for k in range(5):
        ref.set_state(ins[k])
        ref.step(dt)
        assert np.array_equal(outs[k], ref.get_state()), k
