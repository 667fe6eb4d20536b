"""Thin ctypes binding over the C-ABI of include/hydro.h (argument marshalling only).

Every step of the path runs in the CUDA library; nothing here computes.  PyTorch supplies device
memory (its caching allocator is installed as the library's allocator hook) and the stream.
There is no CPU fallback: if the library is not built, or no CUDA device is present, this raises.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

BC_OUTFLOW, BC_REFLECT, BC_PERIODIC, BC_NEIGHBOUR = 0, 1, 2, 3
_ERR = {1: "HYDRO_ERR_ARG", 2: "HYDRO_ERR_ALLOC", 3: "HYDRO_ERR_CUDA", 4: "HYDRO_ERR_UNPHYSICAL",
        5: "HYDRO_ERR_NOSTATE"}

# every symbol include/hydro.h declares (tests check the library exports all of them)
SYMBOLS = ["hydro_create", "hydro_create_nd", "hydro_set_state", "hydro_cfl_dt", "hydro_step", "hydro_evolve",
           "hydro_get_state", "hydro_destroy", "hydro_set_cfl", "hydro_set_limiter_theta",
           "hydro_get_time", "hydro_max_signal_speed", "hydro_set_stream", "hydro_set_allocator",
           "hydro_run_steps", "hydro_ghost_fill", "hydro_get_padded", "hydro_set_kernel_variant",
           "hydro_set_tiling", "hydro_get_tiling", "hydro_tiling_partition", "hydro_set_graph_replay", "hydro_get_axis_order",
           "hydro_create_slab", "hydro_substep", "hydro_halo_count", "hydro_halo_pack",
           "hydro_halo_unpack", "hydro_halo_push", "hydro_state_base", "hydro_smax_device",
           "hydro_reduce_smax", "hydro_host_alloc", "hydro_update_device", "hydro_update_host",
           "hydro_transfer_sync", "hydro_max_signal_speed_noalloc",
           "hydro_set_profiling", "hydro_get_kernel_time", "hydro_launch_count",
           "hydro_is_verification_build", "hydro_last_error"]


class HydroError(RuntimeError):
    def __init__(self, code, where, text=""):
        super().__init__(f"{where}: {_ERR.get(code, code)} {text}".strip())
        self.code = code


_libs = {}
_dp = C.POINTER(C.c_double)
_ALLOC_T = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p)
_FREE_T = C.CFUNCTYPE(None, C.c_void_p)
_hooks = {}


def build(force=False):
    return _build.build(force=force)


def load_library(verify=False):
    """dlopen the production (or -fmad=false verification) library; raises if it is not built."""
    key = bool(verify)
    if key in _libs:
        return _libs[key]
    path = _build.LIB_VERIFY if verify else _build.LIB
    if not os.path.exists(path):
        raise RuntimeError(f"{path} is not built: run `python -m paper_1812_07977_b200.build` "
                           "(there is no CPU fallback)")
    L = C.CDLL(path)
    vp = C.c_void_p
    L.hydro_create.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, C.c_double,
                               C.POINTER(C.c_int), C.POINTER(vp)]
    L.hydro_create_nd.argtypes = [C.c_int, C.POINTER(C.c_int), _dp, C.c_double,
                                  C.POINTER(C.c_int), C.POINTER(vp)]
    L.hydro_set_state.argtypes = [vp, vp]
    L.hydro_get_state.argtypes = [vp, vp]
    L.hydro_get_padded.argtypes = [vp, vp]
    L.hydro_cfl_dt.argtypes = [vp, _dp]
    L.hydro_max_signal_speed.argtypes = [vp, _dp]
    L.hydro_step.argtypes = [vp, C.c_double]
    L.hydro_evolve.argtypes = [vp, C.c_double, C.POINTER(C.c_longlong)]
    L.hydro_destroy.argtypes = [vp]
    L.hydro_set_cfl.argtypes = [vp, C.c_double]
    L.hydro_set_limiter_theta.argtypes = [vp, C.c_double]
    L.hydro_get_time.argtypes = [vp, _dp, C.POINTER(C.c_longlong)]
    L.hydro_set_stream.argtypes = [vp, vp]
    L.hydro_set_allocator.argtypes = [vp, vp]
    L.hydro_run_steps.argtypes = [vp, C.c_longlong]
    L.hydro_ghost_fill.argtypes = [vp]
    L.hydro_set_kernel_variant.argtypes = [vp, C.c_int]
    L.hydro_set_tiling.argtypes = [vp, C.c_int, C.c_int]
    L.hydro_get_tiling.argtypes = [vp, C.POINTER(C.c_int), C.POINTER(C.c_int), C.POINTER(C.c_longlong)]
    L.hydro_set_graph_replay.argtypes = [vp, C.c_int]
    L.hydro_get_axis_order.argtypes = [vp, C.POINTER(C.c_int)]
    L.hydro_tiling_partition.argtypes = [C.c_int] * 8 + [C.POINTER(C.c_int)]
    L.hydro_create_slab.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.POINTER(C.c_int),
                                    C.c_int, C.c_int, C.POINTER(vp), C.POINTER(C.c_int), C.POINTER(C.c_int)]
    L.hydro_substep.argtypes = [vp, C.c_int, C.c_double, C.c_int]
    L.hydro_halo_count.argtypes = [vp, C.POINTER(C.c_size_t)]
    L.hydro_halo_pack.argtypes = [vp, C.c_int, C.c_int, vp]
    L.hydro_halo_unpack.argtypes = [vp, C.c_int, C.c_int, vp]
    L.hydro_halo_push.argtypes = [vp, C.c_int, C.c_int, vp, C.c_int, C.c_longlong]
    L.hydro_state_base.argtypes = [vp, C.c_int, C.POINTER(vp), C.POINTER(C.c_int), C.POINTER(C.c_longlong)]
    L.hydro_smax_device.argtypes = [vp, C.POINTER(vp)]
    L.hydro_reduce_smax.argtypes = [vp]
    L.hydro_host_alloc.argtypes = [vp, C.POINTER(vp)]
    L.hydro_update_device.argtypes = [vp, C.c_uint, vp]
    L.hydro_update_host.argtypes = [vp, C.c_uint, vp]
    L.hydro_transfer_sync.argtypes = [vp]
    L.hydro_max_signal_speed_noalloc.argtypes = [vp, C.c_longlong, C.c_double, vp, vp, vp]
    L.hydro_set_profiling.argtypes = [vp, C.c_int]
    L.hydro_get_kernel_time.argtypes = [vp, C.c_int, _dp, C.POINTER(C.c_longlong)]
    L.hydro_launch_count.restype = C.c_longlong
    L.hydro_is_verification_build.restype = C.c_int
    L.hydro_last_error.restype = C.c_char_p
    _libs[key] = L
    return L


def tiling_partition(nx, ny, nz, tile_rows, planes_per_chunk=0, sms=148, kb=0, ke=None, verify=False):
    """Host logic of the fused kernel's launch geometry (no device needed): the layers of a launch over the
    active planes [kb, ke) as a list of (k0, k1), and the raw (lz, km, nprim, lzr, nlayer)."""
    L = load_library(verify)
    ke = nz if ke is None else ke
    out = (C.c_int * 5)()
    rc = L.hydro_tiling_partition(nx, ny, nz, tile_rows, planes_per_chunk, sms, kb, ke, out)
    if rc:
        raise HydroError(rc, "hydro_tiling_partition", L.hydro_last_error().decode())
    lz, km, nprim, lzr, nlayer = list(out)
    layers = []
    for z in range(nlayer):
        if z < nprim:
            k0 = kb + z * lz; k1 = min(k0 + lz, km)
        else:
            k0 = km + (z - nprim) * lzr; k1 = min(k0 + lzr, ke)
        layers.append((k0, k1))
    return layers, (lz, km, nprim, lzr, nlayer)


NOALLOC_MAX_CELLS = 1 << 27          # HYDRO_NOALLOC_MAX_CELLS


def max_signal_speed_noalloc(U, gamma, smax_out, flag_out, stream=None, verify=False):
    """hydro_max_signal_speed_noalloc: max(|v| + c_s) of a packed CUDA tensor U[5][...] into the CUDA
    tensors smax_out (one float64) and flag_out (one int32), enqueued on `stream` (a cudaStream_t as an
    int; default: torch's current stream).  Allocates nothing; asynchronous."""
    import torch
    L = load_library(verify)
    if not (isinstance(U, torch.Tensor) and U.is_cuda and U.dtype == torch.float64 and U.is_contiguous()
            and U.dim() >= 1 and U.shape[0] == 5):
        raise ValueError("need a contiguous float64 CUDA tensor U[5][...]")
    if not (smax_out.is_cuda and smax_out.dtype == torch.float64 and smax_out.numel() == 1
            and flag_out.is_cuda and flag_out.dtype == torch.int32 and flag_out.numel() == 1):
        raise ValueError("need one float64 and one int32 CUDA element for the outputs")
    if stream is None:
        stream = torch.cuda.current_stream(U.device).cuda_stream
    with torch.cuda.device(U.device):
        rc = L.hydro_max_signal_speed_noalloc(C.c_void_p(U.data_ptr()), U.numel() // 5, float(gamma),
                                              C.c_void_p(smax_out.data_ptr()), C.c_void_p(flag_out.data_ptr()),
                                              C.c_void_p(int(stream)))
    if rc:
        raise HydroError(rc, "hydro_max_signal_speed_noalloc", L.hydro_last_error().decode())


def use_torch_allocator(L, enable=True):
    """Install torch's caching allocator as the library's (process-wide) device-memory hook, or
    restore cudaMalloc / cudaFree with enable=False.  Called around every hydro_create, so that the
    choice is per handle (a handle remembers the release function it was allocated with)."""
    import torch
    key = id(L)
    if not enable:
        rc = L.hydro_set_allocator(None, None)
        if rc:
            raise HydroError(rc, "hydro_set_allocator", L.hydro_last_error().decode())
        return
    if key in _hooks:
        a, f = _hooks[key]
        rc = L.hydro_set_allocator(C.cast(a, C.c_void_p), C.cast(f, C.c_void_p))
        if rc:
            raise HydroError(rc, "hydro_set_allocator", L.hydro_last_error().decode())
        return

    def _alloc(nbytes, stream):
        try:
            return torch.cuda.caching_allocator_alloc(int(nbytes), stream=int(stream or 0))
        except Exception:
            return None

    def _free(ptr):
        try:
            torch.cuda.caching_allocator_delete(int(ptr))
        except Exception:                      # interpreter shutdown: torch is already torn down
            pass

    a, f = _ALLOC_T(_alloc), _FREE_T(_free)
    _hooks[key] = (a, f)                      # keep the callbacks alive
    rc = L.hydro_set_allocator(C.cast(a, C.c_void_p), C.cast(f, C.c_void_p))
    if rc:
        raise HydroError(rc, "hydro_set_allocator", L.hydro_last_error().decode())


def _as_ptr(U, shape, writable=False):
    """(pointer, keepalive, is_device) for a numpy array or a torch tensor of `shape`, fp64."""
    if isinstance(U, np.ndarray):
        if U.dtype != np.float64 or not U.flags.c_contiguous or (writable and not U.flags.writeable):
            raise ValueError("need a C-contiguous float64 array")
        if tuple(U.shape) != tuple(shape):
            raise ValueError(f"shape {U.shape} != {shape}")
        return C.c_void_p(U.ctypes.data), U, False
    import torch
    if isinstance(U, torch.Tensor):
        if U.dtype != torch.float64 or not U.is_contiguous() or tuple(U.shape) != tuple(shape):
            raise ValueError(f"need a contiguous float64 tensor of shape {shape}")
        return C.c_void_p(U.data_ptr()), U, U.is_cuda
    raise TypeError(type(U))


class Hydro:
    """hydro_t with the C-ABI's call names.  `verify=True` loads the -fmad=false build."""

    def __init__(self, nx, ny, nz, gamma, dx, bc, verify=False, torch_allocator=True,
                 stream=None, ndim=None, dxyz=None, slab=None):
        """`slab=(rank, nranks)`: the handle of one z-slab of the global nx*ny*nz grid
        (hydro_create_slab); self.k_first / self.shape then describe the slab."""
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: this library has no CPU fallback")
        self._L = load_library(verify)
        torch.cuda.init()
        use_torch_allocator(self._L, bool(torch_allocator))
        self.shape = (5, nz, ny, nx)
        self._h = C.c_void_p()
        arr = (C.c_int * 6)(*[int(b) for b in bc])
        self.k_first = 0
        if slab is not None:
            k0, nzl = C.c_int(), C.c_int()
            self._chk(self._L.hydro_create_slab(nx, ny, nz, gamma, dx, arr, int(slab[0]), int(slab[1]),
                                                C.byref(self._h), C.byref(k0), C.byref(nzl)), "hydro_create_slab")
            self.k_first, nz = k0.value, nzl.value
            self.shape = (5, nz, ny, nx)
            self.padded_shape = (5, nz + 4, ny + 4, nx + 4)
        elif ndim is None:                                 # 3D run, cubic cells
            self.padded_shape = (5, nz + 4, ny + 4, nx + 4)
            self._chk(self._L.hydro_create(nx, ny, nz, gamma, dx, arr, C.byref(self._h)), "hydro_create")
        else:                                              # run of dimension ndim, cell edges dxyz
            g = [4 if a < ndim else 0 for a in range(3)]
            self.padded_shape = (5, nz + g[2], ny + g[1], nx + g[0])
            n = (C.c_int * 3)(nx, ny, nz)
            d = (C.c_double * 3)(*(dxyz if dxyz is not None else (dx, dx, dx)))
            self._chk(self._L.hydro_create_nd(ndim, n, d, gamma, arr, C.byref(self._h)), "hydro_create_nd")
        # The library enqueues on one stream.  By default that is a torch stream of the handle's own:
        # torch's default stream is the legacy stream 0, which cannot be captured, and
        # hydro_run_steps / hydro_evolve replay a captured CUDA graph.  Device tensors handed to
        # set_state are ordered after the caller's current stream; get_state synchronises.
        if stream is None:
            self.torch_stream = torch.cuda.Stream()
            stream = self.torch_stream.cuda_stream
        else:
            self.torch_stream = torch.cuda.ExternalStream(int(stream)) if int(stream) else torch.cuda.default_stream()
        self._chk(self._L.hydro_set_stream(self._h, C.c_void_p(stream)), "hydro_set_stream")

    def _chk(self, rc, where):
        if rc:
            raise HydroError(rc, where, self._L.hydro_last_error().decode())

    def close(self):
        if getattr(self, "_h", None):
            self._L.hydro_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_cfl(self, cfl):
        self._chk(self._L.hydro_set_cfl(self._h, cfl), "hydro_set_cfl")

    def set_limiter_theta(self, theta):
        self._chk(self._L.hydro_set_limiter_theta(self._h, theta), "hydro_set_limiter_theta")

    def set_kernel_variant(self, variant):
        self._chk(self._L.hydro_set_kernel_variant(self._h, variant), "hydro_set_kernel_variant")

    def set_tiling(self, tile_rows=0, planes_per_chunk=0):
        self._chk(self._L.hydro_set_tiling(self._h, tile_rows, planes_per_chunk), "hydro_set_tiling")

    def get_tiling(self):
        ty, lz, nb = C.c_int(), C.c_int(), C.c_longlong()
        self._chk(self._L.hydro_get_tiling(self._h, C.byref(ty), C.byref(lz), C.byref(nb)),
                  "hydro_get_tiling")
        return {"tile": [32, ty.value], "planes_per_chunk": lz.value, "blocks": nb.value}

    def get_axis_order(self):
        o = (C.c_int * 3)()
        self._chk(self._L.hydro_get_axis_order(self._h, o), "hydro_get_axis_order")
        return list(o)

    def set_graph_replay(self, enable):
        self._chk(self._L.hydro_set_graph_replay(self._h, int(bool(enable))), "hydro_set_graph_replay")

    def set_stream(self, cuda_stream):
        import torch
        self._chk(self._L.hydro_set_stream(self._h, C.c_void_p(cuda_stream)), "hydro_set_stream")
        self.torch_stream = (torch.cuda.ExternalStream(int(cuda_stream)) if int(cuda_stream)
                             else torch.cuda.default_stream())

    def set_state(self, U):
        import torch
        p, keep, on_device = _as_ptr(U, self.shape)
        if on_device:                                  # producer of U ran on the caller's stream
            self.torch_stream.wait_stream(torch.cuda.current_stream())
            U.record_stream(self.torch_stream)
        self._chk(self._L.hydro_set_state(self._h, p), "hydro_set_state")

    def get_state(self, out=None):
        if out is None:
            out = np.empty(self.shape)
        import torch
        p, keep, on_device = _as_ptr(out, self.shape, writable=True)
        if on_device:                                  # earlier users of `out` ran on the caller's stream
            self.torch_stream.wait_stream(torch.cuda.current_stream())
            out.record_stream(self.torch_stream)
        self._chk(self._L.hydro_get_state(self._h, p), "hydro_get_state")   # synchronises
        return out

    def get_padded(self):
        out = np.empty(self.padded_shape)
        self._chk(self._L.hydro_get_padded(self._h, C.c_void_p(out.ctypes.data)), "hydro_get_padded")
        return out

    def ghost_fill(self):
        self._chk(self._L.hydro_ghost_fill(self._h), "hydro_ghost_fill")

    def cfl_dt(self):
        dt = C.c_double()
        self._chk(self._L.hydro_cfl_dt(self._h, C.byref(dt)), "hydro_cfl_dt")
        return dt.value

    def max_signal_speed(self):
        s = C.c_double()
        self._chk(self._L.hydro_max_signal_speed(self._h, C.byref(s)), "hydro_max_signal_speed")
        return s.value

    def step(self, dt):
        self._chk(self._L.hydro_step(self._h, dt), "hydro_step")

    def run_steps(self, n):
        self._chk(self._L.hydro_run_steps(self._h, int(n)), "hydro_run_steps")

    def evolve(self, t_final):
        n = C.c_longlong()
        self._chk(self._L.hydro_evolve(self._h, t_final, C.byref(n)), "hydro_evolve")
        return n.value

    def get_time(self):
        t, n = C.c_double(), C.c_longlong()
        self._chk(self._L.hydro_get_time(self._h, C.byref(t), C.byref(n)), "hydro_get_time")
        return t.value, n.value

    def launch_count(self):
        return self._L.hydro_launch_count()

    # ---- host mirror: selected fields, transfers overlapped with compute ----
    def host_alloc(self):
        """A pinned host array of one packed state, owned by the handle (numpy view)."""
        p = C.c_void_p()
        self._chk(self._L.hydro_host_alloc(self._h, C.byref(p)), "hydro_host_alloc")
        n = int(np.prod(self.shape))
        return np.ctypeslib.as_array(C.cast(p, _dp), shape=(n,)).reshape(self.shape)

    def update_device(self, U_host, fields=31):
        p, keep, on_device = _as_ptr(U_host, self.shape)
        assert not on_device
        self._chk(self._L.hydro_update_device(self._h, fields, p), "hydro_update_device")

    def update_host(self, U_host, fields=31):
        p, keep, on_device = _as_ptr(U_host, self.shape, writable=True)
        assert not on_device
        self._chk(self._L.hydro_update_host(self._h, fields, p), "hydro_update_host")

    def transfer_sync(self):
        self._chk(self._L.hydro_transfer_sync(self._h), "hydro_transfer_sync")

    # ---- z-slab decomposition (driver: paper_1812_07977_b200/slab.py) ----
    def substep(self, stage, dt=0.0, part=0):
        self._chk(self._L.hydro_substep(self._h, stage, dt, part), "hydro_substep")

    def halo_count(self):
        n = C.c_size_t()
        self._chk(self._L.hydro_halo_count(self._h, C.byref(n)), "hydro_halo_count")
        return n.value

    def halo_pack(self, which, side, dst):
        self._chk(self._L.hydro_halo_pack(self._h, which, side, C.c_void_p(dst.data_ptr())), "hydro_halo_pack")

    def halo_unpack(self, which, side, src):
        self._chk(self._L.hydro_halo_unpack(self._h, which, side, C.c_void_p(src.data_ptr())), "hydro_halo_unpack")

    def state_base(self, which):
        p, nz, sv = C.c_void_p(), C.c_int(), C.c_longlong()
        self._chk(self._L.hydro_state_base(self._h, which, C.byref(p), C.byref(nz), C.byref(sv)), "hydro_state_base")
        return p.value, nz.value, sv.value

    def halo_push(self, which, side, peer_base, peer_nz, peer_var_stride):
        self._chk(self._L.hydro_halo_push(self._h, which, side, C.c_void_p(peer_base), peer_nz, peer_var_stride),
                  "hydro_halo_push")

    def smax_device(self):
        p = C.c_void_p()
        self._chk(self._L.hydro_smax_device(self._h, C.byref(p)), "hydro_smax_device")
        return p.value

    def reduce_smax(self):
        self._chk(self._L.hydro_reduce_smax(self._h), "hydro_reduce_smax")
