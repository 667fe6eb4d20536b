"""Axis order (include/hydro.h, hydro_get_axis_order): the library may hold a 3D run of cubic cells with
its axes relabelled when another order tiles better (33 x 257 x 65 -> 257 x 65 x 33).  Nothing a caller
sees may depend on it: states go in and come out in the caller's order, the verification build still
equals the oracle bit for bit (the oracle's association is exactly symmetric under relabelling, pins P4 /
P10), the production build stays within its bars, field masks address the caller's variables."""
import numpy as np
import pytest

from paper_1812_07977_b200 import inputs

pytestmark = pytest.mark.gpu
OUT, REF, PER = 0, 1, 2

# grids with one awkward extent, every boundary kind, the awkward axis first / second
CASES = [((33, 257, 65), (REF, OUT, PER, PER, OUT, REF)),
         ((40, 300, 36), (OUT, OUT, REF, OUT, PER, PER)),
         ((130, 33, 70), (PER, PER, OUT, REF, REF, REF))]


def _gpu(shape, bc, verify, cfl=0.6):
    from paper_1812_07977_b200.binding import Hydro
    g = Hydro(*shape, 1.4, 1.0 / shape[0], bc, verify=verify)
    g.set_cfl(cfl)
    return g


def _cpu(shape, bc, cfl=0.6):
    from oracle import OracleHydro
    c = OracleHydro(*shape, 1.4, 1.0 / shape[0], bc)
    c.set_cfl(cfl)
    return c


@pytest.mark.parametrize("shape,bc", CASES)
def test_relabelled_run_equals_the_oracle(shape, bc):
    import torch
    from test_gpu_parity import assert_one_step_bar
    U = inputs.random_state(*shape, seed=sum(shape), vamp=0.4)
    c = _cpu(shape, bc)
    c.set_state(U)
    g = _gpu(shape, bc, True)
    if torch.cuda.get_device_properties(0).multi_processor_count == 148:
        assert g.get_axis_order() != [0, 1, 2], shape          # these grids are held relabelled on a B200
    g.set_state(U)                                             # from host memory
    assert np.array_equal(g.get_state(), U)
    assert g.max_signal_speed() == c.max_signal_speed()
    for _ in range(3):
        dt = c.cfl_dt()
        assert g.cfl_dt() == dt
        g.step(dt); c.step(dt)
    assert np.array_equal(g.get_state(), c.get_state())
    g.run_steps(3)
    for _ in range(3):
        c.step(c.cfl_dt())
    want = c.get_state()
    assert np.array_equal(g.get_state(), want) and g.get_time() == c.get_time()
    out = torch.empty(g.shape, dtype=torch.float64, device="cuda")
    g.get_state(out)                                           # into device memory
    assert np.array_equal(out.cpu().numpy(), want)
    g.close()
    p = _gpu(shape, bc, False)
    p.set_state(torch.from_numpy(U).cuda())                    # from device memory
    p.run_steps(6)
    assert_one_step_bar(p.get_state(), want, tol=1e-13)
    p.close()


def test_field_masks_address_the_callers_variables_on_a_relabelled_handle():
    from paper_1812_07977_b200.binding import HydroError
    shape, bc = CASES[0]
    U = inputs.random_state(*shape, seed=3)
    V = inputs.random_state(*shape, seed=4)
    g = _gpu(shape, bc, True)
    pin, out = g.host_alloc(), g.host_alloc()
    pin[...] = U
    g.update_device(pin)
    assert np.array_equal(g.get_state(), U)
    pin[...] = V
    g.update_device(pin, fields=2 | 8)                         # m_x and m_z of the caller
    want = U.copy(); want[1] = V[1]; want[3] = V[3]
    assert np.array_equal(g.get_state(), want)
    out[...] = -7.0
    g.update_host(out, fields=4 | 16)                          # m_y and E
    g.transfer_sync()
    assert np.array_equal(out[2], want[2]) and np.array_equal(out[4], want[4])
    assert (out[[0, 1, 3]] == -7.0).all()
    if g.get_axis_order() != [0, 1, 2]:
        with pytest.raises(HydroError):
            g.get_padded()
    g.close()


def test_cubes_and_slabs_keep_their_axes():
    from paper_1812_07977_b200.binding import Hydro
    g = Hydro(64, 64, 64, 1.4, 1.0 / 64, (OUT,) * 6)
    assert g.get_axis_order() == [0, 1, 2]
    g.close()
    g = Hydro(33, 257, 66, 1.4, 1.0 / 33, (OUT,) * 6, slab=(0, 2))
    assert g.get_axis_order() == [0, 1, 2]
    g.close()
    g = Hydro(33, 257, 65, 1.4, 1.0 / 33, (OUT,) * 6, ndim=3, dxyz=(0.1, 0.1, 0.2))   # non-cubic cells
    assert g.get_axis_order() == [0, 1, 2]
    g.close()
