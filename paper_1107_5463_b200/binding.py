"""ctypes binding of libspin (include/spin.h): argument marshalling only.

torch supplies device memory (the workspace tensor) and the CUDA stream; every step of the sweep and of
the measurement runs in the library's kernels.  There is no CPU fallback: importing this module without
a built libspin.so, or creating a system without a CUDA device, raises.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

STORE_INT8, STORE_BITPACK, STORE_FP32, STORE_MSC = 0, 1, 2, 3
J_UNIFORM, J_PER_DIRECTION, J_BOND_PM1 = 0, 1, 2
INIT_HOT, INIT_COLD = 0, 1
OPT_PLAIN_KERNELS = 0
OPT_TMA_KERNELS = 1
OPT_L2_PREFETCH = 2
OPT_KERNEL_VARIANT = 3
OPT_TEMPORAL_BLOCKING = 4
OPT_TBLOCK_ROWS = 5
OPT_L2_KEEP = 6
OPT_DEFER_CAP = 7
UPDATE_METROPOLIS, UPDATE_HEATBATH = 0, 1
_RULE = {"metropolis": UPDATE_METROPOLIS, "heatbath": UPDATE_HEATBATH}
OK, ERR_INVALID_ARG, ERR_UNSUPPORTED, ERR_WORKSPACE_TOO_SMALL, ERR_CUDA, ERR_STATE = range(6)

_STORAGE = {"int8": STORE_INT8, "bitpack": STORE_BITPACK, "fp32": STORE_FP32, "msc": STORE_MSC}
_COUPLING = {"uniform": J_UNIFORM, "per_direction": J_PER_DIRECTION, "bond_pm1": J_BOND_PM1}

# every symbol include/spin.h declares
SYMBOLS = [
    "spin_workspace_bytes", "spin_create", "spin_sweep", "spin_measure", "spin_sweep_record", "spin_sweep_betas", "spin_measure_noalloc", "spin_get_spins",
    "spin_set_spins", "spin_get_spins_device", "spin_set_spins_device", "spin_set_spins_async", "spin_set_spins_status",
    "spin_set_spins_bits_async", "spin_get_spins_bits",
    "spin_get_bonds", "spin_get_sweep_count", "spin_set_sweep_count", "spin_get_launch_count",
    "spin_set_launch_shape", "spin_set_strip_rows", "spin_set_option", "spin_halfsweep", "spin_halo_bytes",
    "spin_halo_get", "spin_halo_put", "spin_halfsweep_range", "spin_halo_pack", "spin_halo_unpack", "spin_halo_wrap", "spin_colour_array", "spin_halo_push", "spin_destroy", "spin_last_error", "spin_version",
]


class SpinConfig(C.Structure):
    _fields_ = [
        ("dims", C.c_int32 * 3), ("n", C.c_int32), ("storage", C.c_int32), ("coupling_kind", C.c_int32),
        ("J", C.c_double * 3), ("bonds", C.c_void_p), ("n_replicas", C.c_int32), ("replica_streams", C.c_int32),
        ("init", C.c_int32), ("seed", C.c_uint64), ("update_rule", C.c_int32),
        ("slab_global", C.c_int32), ("slab_offset", C.c_int32),
    ]


class SpinError(RuntimeError):
    def __init__(self, status, message):
        super().__init__("libspin status %d: %s" % (status, message))
        self.status = status


_lib = None


def lib_path() -> str:
    return _build.LIB


def lib():
    """Load libspin.so (building it if the sources are newer and nvcc is present)."""
    global _lib
    if _lib is None:
        path = _build.LIB
        if _build.is_stale():
            try:
                _build.build()
            except (OSError, FileNotFoundError) as exc:
                if not os.path.exists(path):
                    raise ImportError("libspin.so is not built and nvcc is unavailable: %s" % exc)
        L = C.CDLL(path)
        vp, cfgp = C.c_void_p, C.POINTER(SpinConfig)
        L.spin_workspace_bytes.argtypes = [cfgp, C.POINTER(C.c_size_t)]
        L.spin_create.argtypes = [cfgp, vp, C.c_size_t, vp, C.POINTER(vp)]
        L.spin_sweep.argtypes = [vp, C.c_double, C.c_int64, vp]
        L.spin_measure.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_double), vp]
        L.spin_measure_noalloc.argtypes = [vp, vp, vp, vp]
        L.spin_sweep_betas.argtypes = [vp, C.POINTER(C.c_double), C.c_int64, vp]
        L.spin_sweep_record.argtypes = [vp, C.c_double, C.c_int64, vp, vp, vp]
        L.spin_get_spins.argtypes = [vp, vp, C.c_size_t]
        L.spin_set_spins.argtypes = [vp, vp, C.c_size_t]
        L.spin_get_spins_device.argtypes = [vp, vp, C.c_size_t, vp]
        L.spin_set_spins_device.argtypes = [vp, vp, C.c_size_t, vp, vp]
        L.spin_set_spins_async.argtypes = [vp, vp, C.c_size_t, vp]
        L.spin_set_spins_status.argtypes = [vp, vp]
        L.spin_set_spins_bits_async.argtypes = [vp, vp, C.c_size_t, vp]
        L.spin_get_spins_bits.argtypes = [vp, vp, C.c_size_t, vp]
        L.spin_get_bonds.argtypes = [vp, vp, C.c_size_t]
        L.spin_get_sweep_count.argtypes = [vp, C.POINTER(C.c_uint64)]
        L.spin_set_sweep_count.argtypes = [vp, C.c_uint64]
        L.spin_get_launch_count.argtypes = [vp, C.POINTER(C.c_uint64)]
        L.spin_set_launch_shape.argtypes = [vp, C.c_int32, C.c_int32, C.c_int32]
        L.spin_set_strip_rows.argtypes = [vp, C.c_int32]
        L.spin_set_option.argtypes = [vp, C.c_int32, C.c_int64]
        L.spin_halfsweep.argtypes = [vp, C.c_double, C.c_int32, vp]
        L.spin_halo_bytes.argtypes = [vp, C.POINTER(C.c_size_t)]
        L.spin_halo_get.argtypes = [vp, C.c_int32, C.c_int32, vp, vp]
        L.spin_halo_put.argtypes = [vp, C.c_int32, C.c_int32, vp, vp]
        L.spin_halfsweep_range.argtypes = [vp, C.c_double, C.c_int32, C.c_int32, C.c_int32, C.c_int32, vp]
        L.spin_halo_pack.argtypes = [vp, C.c_int32, vp, vp]
        L.spin_halo_unpack.argtypes = [vp, C.c_int32, vp, vp]
        L.spin_halo_wrap.argtypes = [vp, C.c_int32, vp]
        L.spin_colour_array.argtypes = [vp, C.c_int32, C.POINTER(vp), C.POINTER(C.c_size_t)]
        L.spin_halo_push.argtypes = [vp, C.c_int32, vp, vp, vp]
        L.spin_destroy.argtypes = [vp]
        for name in SYMBOLS:
            getattr(L, name).restype = C.c_int
        L.spin_last_error.restype = C.c_char_p
        L.spin_last_error.argtypes = []
        L.spin_version.restype = C.c_char_p
        L.spin_version.argtypes = []
        _lib = L
    return _lib


def _check(status):
    if status != OK:
        raise SpinError(status, lib().spin_last_error().decode())


def make_config(dims, n=1, storage="int8", coupling="uniform", J=(1.0, 1.0, 1.0), bonds=None, replicas=1,
                replica_streams=0, init=INIT_HOT, seed=0, rule="metropolis", slab_global=0, slab_offset=0):
    dims = [int(v) for v in dims]
    if len(dims) == 2:
        dims.append(1)
    cfg = SpinConfig()
    cfg.dims[:] = dims
    cfg.n = int(n)
    cfg.storage = _STORAGE[storage] if isinstance(storage, str) else int(storage)
    cfg.coupling_kind = _COUPLING[coupling] if isinstance(coupling, str) else int(coupling)
    Jv = [float(v) for v in (J if hasattr(J, "__len__") else (J, J, J))]
    while len(Jv) < 3:
        Jv.append(0.0)
    cfg.J[:] = Jv
    keep = None
    if bonds is not None:
        keep = np.ascontiguousarray(bonds, dtype=np.int8)
        cfg.bonds = keep.ctypes.data
    else:
        cfg.bonds = None
    cfg.n_replicas = int(replicas)
    cfg.replica_streams = int(replica_streams)
    cfg.init = int(init)
    cfg.seed = int(seed)
    cfg.update_rule = _RULE[rule] if isinstance(rule, str) else int(rule)
    cfg.slab_global = int(slab_global)
    cfg.slab_offset = int(slab_offset)
    return cfg, keep


def workspace_bytes(cfg) -> int:
    out = C.c_size_t(0)
    _check(lib().spin_workspace_bytes(C.byref(cfg), C.byref(out)))
    return int(out.value)


class SpinSystem:
    """One lattice system on the current CUDA device.  Same names as the C ABI: sweep, measure,
    sweep_record, get_spins, set_spins, get_bonds."""

    def __init__(self, dims, n=1, storage="int8", coupling="uniform", J=(1.0, 1.0, 1.0), bonds=None, replicas=1,
                 replica_streams=0, init=INIT_HOT, seed=0, device="cuda:0", rule="metropolis", slab_global=0,
                 slab_offset=0):
        import torch

        if not torch.cuda.is_available():
            raise RuntimeError("libspin needs a CUDA device (there is no CPU fallback)")
        self._torch = torch
        self.device = torch.device(device)
        cfg, keep = make_config(dims, n, storage, coupling, J, bonds, replicas, replica_streams, init, seed, rule,
                                slab_global, slab_offset)
        self.cfg = cfg
        self.dims = tuple(cfg.dims)
        self.n = int(cfg.n)
        self.R = int(cfg.n_replicas)
        self.N = self.dims[0] * self.dims[1] * self.dims[2]
        self.d = 2 if self.dims[2] == 1 else 3
        self._h = None
        nbytes = workspace_bytes(cfg)
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            base = self.workspace.data_ptr()
            self._ws_ptr = (base + 255) & ~255
            h = C.c_void_p()
            _check(lib().spin_create(C.byref(cfg), C.c_void_p(self._ws_ptr), nbytes, self._stream(), C.byref(h)))
        self._h = h
        del keep

    def _stream(self):
        return C.c_void_p(self._torch.cuda.current_stream(self.device).cuda_stream)

    def close(self):
        if getattr(self, "_h", None):
            lib().spin_destroy(self._h)
            self._h = None

    __del__ = close

    def sweep(self, beta, n_sweeps=1):
        with self._torch.cuda.device(self.device):
            _check(lib().spin_sweep(self._h, float(beta), int(n_sweeps), self._stream()))

    def sweep_betas(self, betas, n_sweeps=1):
        """temperature axis: replica r at betas[r]"""
        b = np.ascontiguousarray(betas, dtype=np.float64)
        if b.shape != (self.R,):
            raise ValueError("betas must hold one value per replica")
        with self._torch.cuda.device(self.device):
            _check(lib().spin_sweep_betas(self._h, b.ctypes.data_as(C.POINTER(C.c_double)), int(n_sweeps), self._stream()))

    def halfsweep(self, beta, colour):
        with self._torch.cuda.device(self.device):
            _check(lib().spin_halfsweep(self._h, float(beta), int(colour), self._stream()))

    def halfsweep_range(self, beta, colour, plane0, n_planes, last):
        with self._torch.cuda.device(self.device):
            _check(lib().spin_halfsweep_range(self._h, float(beta), int(colour), int(plane0), int(n_planes), int(bool(last)), self._stream()))

    def halo_pack(self, colour, buf):
        """both owned boundary planes of colour `colour` -> buf (CUDA uint8 tensor of 2 * halo_bytes: [lowest][highest])"""
        with self._torch.cuda.device(self.device):
            _check(lib().spin_halo_pack(self._h, int(colour), C.c_void_p(buf.data_ptr()), self._stream()))

    def halo_unpack(self, colour, buf):
        """buf = [plane from the slab below][plane from the slab above] -> the two ghost planes"""
        with self._torch.cuda.device(self.device):
            _check(lib().spin_halo_unpack(self._h, int(colour), C.c_void_p(buf.data_ptr()), self._stream()))

    def colour_array(self, colour):
        """(device address, bytes) of the colour array: what a neighbouring slab's owner maps for peer stores"""
        ptr, n = C.c_void_p(), C.c_size_t(0)
        _check(lib().spin_colour_array(self._h, int(colour), C.byref(ptr), C.byref(n)))
        return int(ptr.value), int(n.value)

    def halo_push(self, colour, peer_below_ptr, peer_above_ptr):
        """my two owned boundary planes -> the ghost planes of the slabs below and above (peer stores, one kernel)"""
        with self._torch.cuda.device(self.device):
            _check(lib().spin_halo_push(self._h, int(colour), C.c_void_p(peer_below_ptr), C.c_void_p(peer_above_ptr), self._stream()))

    def halo_wrap(self, colour):
        """single slab, periodic: its own boundary planes become its ghost planes (one kernel)"""
        with self._torch.cuda.device(self.device):
            _check(lib().spin_halo_wrap(self._h, int(colour), self._stream()))

    def halo_bytes(self):
        out = C.c_size_t(0)
        _check(lib().spin_halo_bytes(self._h, C.byref(out)))
        return int(out.value)

    def halo_get(self, colour, side, buf):
        """owned boundary plane (side 0: lowest, 1: highest) of colour `colour` -> contiguous CUDA uint8 tensor buf"""
        with self._torch.cuda.device(self.device):
            _check(lib().spin_halo_get(self._h, int(colour), int(side), C.c_void_p(buf.data_ptr()), self._stream()))

    def halo_put(self, colour, side, buf):
        """contiguous CUDA uint8 tensor buf -> ghost plane below (side 0) / above (side 1) the owned planes"""
        with self._torch.cuda.device(self.device):
            _check(lib().spin_halo_put(self._h, int(colour), int(side), C.c_void_p(buf.data_ptr()), self._stream()))

    def measure(self):
        E = np.zeros(self.R, dtype=np.float64)
        M = np.zeros(self.R * self.n, dtype=np.float64)
        dp = C.POINTER(C.c_double)
        with self._torch.cuda.device(self.device):
            _check(lib().spin_measure(self._h, E.ctypes.data_as(dp), M.ctypes.data_as(dp), self._stream()))
        return E, M.reshape(self.R, self.n)

    def measure_noalloc(self, d_E, d_M):
        """E, M into the caller's CUDA float64 tensors d_E [R], d_M [R, n]; asynchronous, allocates nothing (the scratch is a
        fixed array inside the library: spin.h)"""
        with self._torch.cuda.device(self.device):
            _check(lib().spin_measure_noalloc(self._h, C.c_void_p(d_E.data_ptr()), C.c_void_p(d_M.data_ptr()), self._stream()))

    def sweep_record(self, beta, n_sweeps, d_E=None, d_M=None):
        """Returns (d_E, d_M): CUDA float64 tensors [n_sweeps, R] and [n_sweeps, R, n] (filled asynchronously)."""
        torch = self._torch
        if d_E is None:
            d_E = torch.empty((int(n_sweeps), self.R), dtype=torch.float64, device=self.device)
        if d_M is None:
            d_M = torch.empty((int(n_sweeps), self.R, self.n), dtype=torch.float64, device=self.device)
        with torch.cuda.device(self.device):
            _check(lib().spin_sweep_record(self._h, float(beta), int(n_sweeps), C.c_void_p(d_E.data_ptr()),
                                           C.c_void_p(d_M.data_ptr()), self._stream()))
        return d_E, d_M

    def get_spins(self):
        out = (np.empty((self.R, self.N), dtype=np.int8) if self.n == 1
               else np.empty((self.R, self.N, self.n), dtype=np.float32))
        with self._torch.cuda.device(self.device):
            _check(lib().spin_get_spins(self._h, out.ctypes.data_as(C.c_void_p), out.nbytes))
        return out

    def set_spins(self, spins):
        a = np.ascontiguousarray(spins, dtype=np.int8 if self.n == 1 else np.float32)
        with self._torch.cuda.device(self.device):
            _check(lib().spin_set_spins(self._h, a.ctypes.data_as(C.c_void_p), a.nbytes))

    def set_spins_async(self, spins):
        """host array (pinned: truly asynchronous) -> arrays on the current stream; set_spins_status() reports the +-1 check"""
        a = np.ascontiguousarray(spins, dtype=np.int8 if self.n == 1 else np.float32)
        self._pending_host = a          # must stay valid until the stream has consumed it
        with self._torch.cuda.device(self.device):
            _check(lib().spin_set_spins_async(self._h, a.ctypes.data_as(C.c_void_p), a.nbytes, self._stream()))

    def set_spins_status(self):
        with self._torch.cuda.device(self.device):
            _check(lib().spin_set_spins_status(self._h, self._stream()))
        self._pending_host = None

    def set_spins_bits_async(self, bits):
        """canonical bit array (uint8 [R, N / 8], bit (i & 7) of byte i >> 3 set = spin -1; np.packbits(s < 0, bitorder="little"))
        -> arrays on the current stream"""
        a = np.ascontiguousarray(bits, dtype=np.uint8)
        self._pending_host = a
        with self._torch.cuda.device(self.device):
            _check(lib().spin_set_spins_bits_async(self._h, a.ctypes.data_as(C.c_void_p), a.nbytes, self._stream()))

    def get_spins_bits(self):
        out = np.empty((self.R, self.N // 8), dtype=np.uint8)
        with self._torch.cuda.device(self.device):
            _check(lib().spin_get_spins_bits(self._h, out.ctypes.data_as(C.c_void_p), out.nbytes, self._stream()))
        return out

    def get_spins_device(self, out=None):
        """canonical spins as a CUDA tensor (int8 [R, N] or float32 [R, N, n]), converted on the current stream"""
        torch = self._torch
        if out is None:
            out = (torch.empty((self.R, self.N), dtype=torch.int8, device=self.device) if self.n == 1
                   else torch.empty((self.R, self.N, self.n), dtype=torch.float32, device=self.device))
        with torch.cuda.device(self.device):
            _check(lib().spin_get_spins_device(self._h, C.c_void_p(out.data_ptr()), out.numel() * out.element_size(), self._stream()))
        return out

    def set_spins_device(self, canon):
        """canonical spins from a contiguous CUDA tensor; returns the device flag tensor of the +-1 check (n = 1) or None"""
        torch = self._torch
        flag = torch.zeros(1, dtype=torch.int32, device=self.device) if self.n == 1 else None
        with torch.cuda.device(self.device):
            _check(lib().spin_set_spins_device(self._h, C.c_void_p(canon.data_ptr()), canon.numel() * canon.element_size(),
                                               C.c_void_p(flag.data_ptr()) if flag is not None else None, self._stream()))
        return flag

    def get_bonds(self):
        out = np.empty((self.R, self.d, self.N), dtype=np.int8)
        with self._torch.cuda.device(self.device):
            _check(lib().spin_get_bonds(self._h, out.ctypes.data_as(C.c_void_p), out.nbytes))
        return out

    @property
    def sweep_counter(self):
        t = C.c_uint64(0)
        _check(lib().spin_get_sweep_count(self._h, C.byref(t)))
        return int(t.value)

    @sweep_counter.setter
    def sweep_counter(self, t):
        _check(lib().spin_set_sweep_count(self._h, int(t)))

    @property
    def launch_count(self):
        t = C.c_uint64(0)
        _check(lib().spin_get_launch_count(self._h, C.byref(t)))
        return int(t.value)

    def set_launch_shape(self, block=0, grid_num=1, grid_den=1):
        _check(lib().spin_set_launch_shape(self._h, int(block), int(grid_num), int(grid_den)))

    def set_strip_rows(self, rows=0):
        _check(lib().spin_set_strip_rows(self._h, int(rows)))

    def set_option(self, option, value):
        _check(lib().spin_set_option(self._h, int(option), int(value)))


def from_workload(w, seed, **over):
    """Build a SpinSystem from a workloads.WORKLOADS recipe."""
    kw = dict(dims=w["dims"], n=w["n"], storage=w["storage"], coupling=w["coupling"], J=w["J"],
              replicas=w["replicas"], replica_streams=w["replica_streams"], seed=seed)
    kw.update(over)
    return SpinSystem(**kw)
