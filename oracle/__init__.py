"""CPU oracle for the checkerboard Metropolis sweep -- TEST INFRASTRUCTURE, NOT PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It never imports the CUDA binding
(paper_1107_5463_b200) and shares no code with it.  All arithmetic lives in
oracle/spin_oracle.cpp (plain single-threaded C++); this file is a ctypes
marshalling layer only.
"""
import ctypes as C

import numpy as np

from . import build as _build

J_UNIFORM, J_PER_DIRECTION, J_BOND_PM1 = 0, 1, 2
INIT_HOT, INIT_COLD = 0, 1
RULE_METROPOLIS, RULE_HEATBATH = 0, 1

_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        u32p = C.POINTER(C.c_uint32)
        L.oracle_philox4x32_10.argtypes = [u32p, u32p, u32p]
        L.oracle_philox4x32_10.restype = None
        L.oracle_rand.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32, u32p]
        L.oracle_rand.restype = None
        L.oracle_vector_site_words.argtypes = [C.c_uint64, C.c_int, C.c_int, C.c_uint64, C.c_uint32, C.c_uint32, C.c_int, u32p]
        L.oracle_vector_site_words.restype = None
        L.oracle_ising_uniform.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32, C.c_uint32, C.c_int]
        L.oracle_ising_uniform.restype = C.c_uint32
        L.oracle_threshold.argtypes = [C.c_double, C.c_int]
        L.oracle_threshold.restype = C.c_uint64
        L.oracle_ising_accept.argtypes = [C.c_double, C.c_int, C.c_uint32]
        L.oracle_ising_accept.restype = C.c_int
        L.oracle_u24.argtypes = [C.c_uint32]
        L.oracle_u24.restype = C.c_float
        L.oracle_direction3.argtypes = [C.c_uint32, C.c_uint32, C.POINTER(C.c_float)]
        L.oracle_direction3.restype = None
        L.oracle_direction2.argtypes = [C.c_uint32, C.POINTER(C.c_float)]
        L.oracle_direction2.restype = None
        L.oracle_vector_accept.argtypes = [C.c_double, C.c_float, C.c_uint32]
        L.oracle_vector_accept.restype = C.c_int
        L.oracle_create.argtypes = [C.POINTER(C.c_int32), C.c_int32, C.c_int32, C.POINTER(C.c_double), C.c_void_p,
                                    C.c_int32, C.c_int32, C.c_int32, C.c_uint64]
        L.oracle_create.restype = C.c_void_p
        L.oracle_set_update_rule.argtypes = [C.c_void_p, C.c_int32]
        L.oracle_set_update_rule.restype = C.c_int
        L.oracle_heatbath_threshold.argtypes = [C.c_double, C.c_int]
        L.oracle_heatbath_threshold.restype = C.c_uint64
        L.oracle_heatbath3.argtypes = [C.c_double, C.POINTER(C.c_float), C.c_uint32, C.c_uint32, C.POINTER(C.c_float)]
        L.oracle_heatbath3.restype = None
        L.oracle_destroy.argtypes = [C.c_void_p]
        L.oracle_destroy.restype = None
        L.oracle_sweep.argtypes = [C.c_void_p, C.c_double, C.c_int64]
        L.oracle_sweep.restype = C.c_int
        L.oracle_sweep_count.argtypes = [C.c_void_p, C.c_double, C.c_int64, C.POINTER(C.c_int64)]
        L.oracle_sweep_count.restype = C.c_int
        L.oracle_last_sweep_dE.argtypes = [C.c_void_p]
        L.oracle_last_sweep_dE.restype = C.c_double
        L.oracle_measure.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.oracle_measure.restype = C.c_int
        L.oracle_get_spins.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64]
        L.oracle_get_spins.restype = C.c_int
        L.oracle_set_spins.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64]
        L.oracle_set_spins.restype = C.c_int
        L.oracle_get_bonds.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64]
        L.oracle_get_bonds.restype = C.c_int
        L.oracle_get_sweep_count.argtypes = [C.c_void_p]
        L.oracle_get_sweep_count.restype = C.c_uint64
        L.oracle_set_sweep_count.argtypes = [C.c_void_p, C.c_uint64]
        L.oracle_set_sweep_count.restype = None
        _lib = L
    return _lib


def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*[int(v) & 0xFFFFFFFF for v in ctr])
    k = (C.c_uint32 * 2)(*[int(v) & 0xFFFFFFFF for v in key])
    o = (C.c_uint32 * 4)()
    lib().oracle_philox4x32_10(c, k, o)
    return [int(v) for v in o]


def rand(seed, unit, rho, t, tag):
    o = (C.c_uint32 * 4)()
    lib().oracle_rand(seed, unit, rho, t, tag, o)
    return [int(v) for v in o]


def vector_site_words(seed, n, j, rho, t, colour, rule=0):
    """words of the n >= 2 update of the site with compressed index j (n = 2 and heat bath: pairs of sites share a call, R-16b)"""
    o = (C.c_uint32 * 4)()
    lib().oracle_vector_site_words(seed, n, rule, j, rho, t, colour, o)
    return [int(v) for v in o]


def ising_uniform(seed, j, rho, t, colour):
    return int(lib().oracle_ising_uniform(seed, j, rho, t, colour))


def threshold(beta, dE):
    return int(lib().oracle_threshold(float(beta), int(dE)))


def ising_accept(beta, dE, U):
    return int(lib().oracle_ising_accept(float(beta), int(dE), int(U)))


def u24(w):
    return float(lib().oracle_u24(int(w)))


def direction3(a, b):
    o = (C.c_float * 3)()
    lib().oracle_direction3(int(a), int(b), o)
    return np.array(list(o), dtype=np.float32)


def direction2(a):
    o = (C.c_float * 2)()
    lib().oracle_direction2(int(a), o)
    return np.array(list(o), dtype=np.float32)


def vector_accept(beta, dE, w):
    return int(lib().oracle_vector_accept(float(beta), float(np.float32(dE)), int(w)))


def heatbath_threshold(beta, h):
    return int(lib().oracle_heatbath_threshold(float(beta), int(h)))


def heatbath3(beta, h, w0, w1):
    hv = (C.c_float * 3)(*[float(np.float32(v)) for v in h])
    o = (C.c_float * 3)()
    lib().oracle_heatbath3(float(beta), hv, int(w0), int(w1), o)
    return np.array(list(o), dtype=np.float32)


class System:
    """One oracle lattice system (R replicas).  Mirrors the product's handle, separately implemented."""

    def __init__(self, dims, n=1, coupling_kind=J_UNIFORM, J=(1.0, 1.0, 1.0), bonds=None, n_replicas=1,
                 replica_streams=0, init=INIT_HOT, seed=0, rule=RULE_METROPOLIS):
        dims = [int(v) for v in dims]
        if len(dims) == 2:
            dims = dims + [1]
        self.dims = tuple(dims)
        self.n = int(n)
        self.R = int(n_replicas)
        self.N = dims[0] * dims[1] * dims[2]
        self.d = 2 if dims[2] == 1 else 3
        self.coupling_kind = coupling_kind
        cd = (C.c_int32 * 3)(*dims)
        Jv = list(J) if hasattr(J, "__len__") else [J, J, J]
        while len(Jv) < 3:
            Jv.append(0.0)
        cJ = (C.c_double * 3)(*[float(v) for v in Jv])
        bptr = None
        if bonds is not None:
            self._bonds_in = np.ascontiguousarray(bonds, dtype=np.int8)
            assert self._bonds_in.size == self.R * self.d * self.N
            bptr = self._bonds_in.ctypes.data_as(C.c_void_p)
        self._h = lib().oracle_create(cd, self.n, coupling_kind, cJ, bptr, self.R, int(replica_streams), int(init),
                                      int(seed))
        if not self._h:
            raise ValueError("oracle_create: invalid arguments")
        if rule != RULE_METROPOLIS and lib().oracle_set_update_rule(self._h, int(rule)):
            raise ValueError("oracle_set_update_rule: rule not offered for this model")

    def close(self):
        if getattr(self, "_h", None):
            lib().oracle_destroy(self._h)
            self._h = None

    __del__ = close

    def sweep(self, beta, n_sweeps=1):
        rc = lib().oracle_sweep(self._h, float(beta), int(n_sweeps))
        if rc:
            raise RuntimeError("oracle_sweep failed (%d)" % rc)

    def sweep_count(self, beta, n_sweeps=1):
        acc = np.zeros(int(n_sweeps), dtype=np.int64)
        rc = lib().oracle_sweep_count(self._h, float(beta), int(n_sweeps), acc.ctypes.data_as(C.POINTER(C.c_int64)))
        if rc:
            raise RuntimeError("oracle_sweep_count failed (%d)" % rc)
        return acc

    def last_sweep_dE(self):
        """Sum of the dE of every move accepted in the last Metropolis sweep (bookkeeping)."""
        return float(lib().oracle_last_sweep_dE(self._h))

    def measure(self):
        E = np.zeros(self.R, dtype=np.float64)
        M = np.zeros(self.R * self.n, dtype=np.float64)
        rc = lib().oracle_measure(self._h, E.ctypes.data_as(C.POINTER(C.c_double)),
                                  M.ctypes.data_as(C.POINTER(C.c_double)))
        if rc:
            raise RuntimeError("oracle_measure failed")
        return E, M.reshape(self.R, self.n)

    def get_spins(self):
        if self.n == 1:
            out = np.empty((self.R, self.N), dtype=np.int8)
        else:
            out = np.empty((self.R, self.N, self.n), dtype=np.float32)
        rc = lib().oracle_get_spins(self._h, out.ctypes.data_as(C.c_void_p), out.nbytes)
        if rc:
            raise RuntimeError("oracle_get_spins failed")
        return out

    def set_spins(self, spins):
        dt = np.int8 if self.n == 1 else np.float32
        a = np.ascontiguousarray(spins, dtype=dt)
        rc = lib().oracle_set_spins(self._h, a.ctypes.data_as(C.c_void_p), a.nbytes)
        if rc:
            raise ValueError("oracle_set_spins: bad size or values")

    def get_bonds(self):
        out = np.empty((self.R, self.d, self.N), dtype=np.int8)
        rc = lib().oracle_get_bonds(self._h, out.ctypes.data_as(C.c_void_p), out.nbytes)
        if rc:
            raise RuntimeError("oracle_get_bonds failed")
        return out

    @property
    def sweep_counter(self):
        return int(lib().oracle_get_sweep_count(self._h))

    @sweep_counter.setter
    def sweep_counter(self, t):
        lib().oracle_set_sweep_count(self._h, int(t))
