"""ctypes wrapper around oracle/smcx_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
import this package.  It imports nothing from paper_2509_20949_b200.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "smcx_oracle.cpp")
_LIB = os.path.join(_HERE, "libsmcx_oracle.so")
_lock = threading.Lock()
_lib = None

BCC, FCC = 0, 1


def build(force: bool = False) -> str:
    """g++ -O2 the oracle into oracle/libsmcx_oracle.so (rebuilt when the source is newer)."""
    with _lock:
        stale = (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC)
        if force or stale:
            tmp = _LIB + f".tmp{os.getpid()}"
            subprocess.check_call(
                ["g++", "-O2", "-std=c++17", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra", "-o", tmp, _SRC])
            os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is not None:
        return _lib
    lib = C.CDLL(build())
    u32p, i32p, i64p = C.POINTER(C.c_uint32), C.POINTER(C.c_int32), C.POINTER(C.c_int64)
    u8p, f64p = C.POINTER(C.c_uint8), C.POINTER(C.c_double)
    sig = {
        "oracle_philox4x32_10": (None, [u32p, u32p, u32p]),
        "oracle_shell": (C.c_int, [C.c_int, C.c_int, i32p, C.c_int]),
        "oracle_create": (C.c_void_p, [C.c_int, i32p, C.c_int, C.c_int, i32p, C.c_int, u32p, C.c_int,
                                       C.c_uint64]),
        "oracle_destroy": (None, [C.c_void_p]),
        "oracle_set_local_model": (None, [C.c_void_p, i32p]),
        "oracle_site_energy": (C.c_int64, [C.c_void_p, C.c_int64]),
        "oracle_n_sites": (C.c_int64, [C.c_void_p]),
        "oracle_init_species": (None, [C.c_void_p]),
        "oracle_init_permutation": (C.c_uint64, [C.c_void_p, C.c_uint64]),
        "oracle_init_composition": (C.c_int, [C.c_void_p, C.POINTER(C.c_int64)]),
        "oracle_set_species": (C.c_int, [C.c_void_p, u8p]),
        "oracle_get_species": (None, [C.c_void_p, u8p]),
        "oracle_set_temperature": (None, [C.c_void_p, u32p, C.c_int]),
        "oracle_energy": (C.c_int64, [C.c_void_p]),
        "oracle_running_energy": (C.c_int64, [C.c_void_p]),
        "oracle_neighbour": (C.c_int64, [C.c_void_p, C.c_int64, C.c_int, C.c_int]),
        "oracle_delta_e": (C.c_int64, [C.c_void_p, C.c_int64, C.c_int]),
        "oracle_lc_valid": (C.c_int, [C.c_void_p]),
        "oracle_sweep_lc": (C.c_int, [C.c_void_p, C.c_int64, C.c_int, C.c_uint32]),
        "oracle_sweep_seq": (None, [C.c_void_p, C.c_int64]),
        "oracle_sweep_lc_slabs": (C.c_int64, [C.c_void_p, C.c_int64, C.c_int, C.c_int, C.c_int, C.c_uint32]),
        "oracle_slab_partition": (C.c_int, [C.c_void_p, C.c_int, i32p]),
        "oracle_set_threads": (C.c_int, [C.c_void_p, C.c_int]),
        "oracle_shift": (None, [C.c_void_p, C.c_uint32, i32p]),
        "oracle_stats": (None, [C.c_void_p, i64p, i64p, i64p]),
        "oracle_trace": (C.c_int64, [C.c_void_p, C.c_int64, C.c_int64, i64p]),
        "oracle_set_sweep_counter": (C.c_int, [C.c_void_p, C.c_int64]),
        "oracle_count_visits": (None, [C.c_void_p, C.c_int]),
        "oracle_get_visits": (None, [C.c_void_p, u32p]),
        "oracle_pair_counts": (None, [C.c_void_p, i64p]),
        "oracle_sro": (None, [C.c_void_p, f64p, i64p]),
        "oracle_exchange_delta": (C.c_double, [C.c_int64, C.c_int64, C.c_int32, C.c_int32]),
        "oracle_exchange_accept": (C.c_int, [C.c_int64, C.c_int64, C.c_int32, C.c_int32, C.c_uint32]),
        "oracle_exchange_draw": (C.c_uint32, [C.c_uint64, C.c_uint64, C.c_uint32]),
    }
    for name, (res, args) in sig.items():
        fn = getattr(lib, name)
        fn.restype = res
        fn.argtypes = args
    _lib = lib
    return lib


def _ptr(a: np.ndarray, ctype):
    return a.ctypes.data_as(C.POINTER(ctype))


def philox4x32_10(ctr, key):
    lib = _load()
    c = np.asarray(ctr, dtype=np.uint32).copy()
    k = np.asarray(key, dtype=np.uint32).copy()
    out = np.zeros(4, dtype=np.uint32)
    lib.oracle_philox4x32_10(_ptr(c, C.c_uint32), _ptr(k, C.c_uint32), _ptr(out, C.c_uint32))
    return tuple(int(v) for v in out)


def shell(lattice: int, s: int) -> np.ndarray:
    """Offsets (dx,dy,dz) of neighbour shell s in half-lattice units, in the oracle's order."""
    lib = _load()
    buf = np.zeros((512, 3), dtype=np.int32)
    n = lib.oracle_shell(lattice, s, _ptr(buf, C.c_int32), 512)
    return buf[:n].copy()


def exchange_delta(E_i: int, E_j: int, kT_i: int, kT_j: int) -> float:
    """Delta of Eq. 6 for integer energies and temperatures in 0.1 meV."""
    return float(_load().oracle_exchange_delta(int(E_i), int(E_j), int(kT_i), int(kT_j)))


def exchange_accept(E_i: int, E_j: int, kT_i: int, kT_j: int, u: int) -> bool:
    """Eq. 5 in integer form: accept iff Delta >= 0 or u < floor(exp(Delta) 2^32)."""
    return bool(_load().oracle_exchange_accept(int(E_i), int(E_j), int(kT_i), int(kT_j), int(u)))


def exchange_draw(seed: int, rnd: int, p: int) -> int:
    return int(_load().oracle_exchange_draw(C.c_uint64(int(seed)), C.c_uint64(int(rnd)), int(p)))


def replica_exchange(replicas: list, kT: list, tables: list, parity: int, seed: int, rnd: int,
                     energy=lambda o: o.running_energy()) -> list:
    """One round of replica exchange (S9; Eq. 5-6) over temperature slots.

    ``replicas[p]`` is the Oracle running at slot p (temperature ``kT[p]``, threshold table
    ``tables[p]``).  Slots p, p + 1 with p = parity, parity + 2, ... attempt an exchange; when it is
    accepted the two configurations change slots (the list is permuted in place and each Oracle is
    given the table of its new slot).  Returns the list of accept flags, one per slot pair (0 for the
    pairs not attempted in this round).
    """
    n = len(replicas)
    flags = [0] * max(0, n - 1)
    for p in range(parity & 1, n - 1, 2):
        u = exchange_draw(seed, rnd, p)
        if exchange_accept(energy(replicas[p]), energy(replicas[p + 1]), kT[p], kT[p + 1], u):
            replicas[p], replicas[p + 1] = replicas[p + 1], replicas[p]
            replicas[p].set_temperature(tables[p])
            replicas[p + 1].set_temperature(tables[p + 1])
            flags[p] = 1
    return flags


class Oracle:
    """One lattice + schedule state.  Method names follow include/smcx.h where they overlap."""

    def __init__(self, lattice, dims, n_species, n_shells, epi, link_cell, accept, seed,
                 init: bool = True, threads: int = 1):
        lib = _load()
        self._lib = lib
        self.lattice, self.dims = int(lattice), tuple(int(d) for d in dims)
        self.n_species, self.n_shells = int(n_species), int(n_shells)
        epi = np.ascontiguousarray(epi, dtype=np.int32)
        assert epi.shape == (n_shells, n_species, n_species)
        accept = np.ascontiguousarray(accept, dtype=np.uint32)
        d = np.asarray(self.dims, dtype=np.int32)
        self._h = lib.oracle_create(self.lattice, _ptr(d, C.c_int32), self.n_species, self.n_shells,
                                    _ptr(epi, C.c_int32), int(link_cell), _ptr(accept, C.c_uint32),
                                    int(accept.size), C.c_uint64(int(seed)))
        if not self._h:
            raise ValueError("oracle_create rejected the parameters")
        self.n_sites = int(lib.oracle_n_sites(self._h))
        self.threads = int(lib.oracle_set_threads(self._h, int(threads)))
        if init:
            lib.oracle_init_species(self._h)

    @classmethod
    def from_config(cls, cfg, init: bool = True, threads: int = 1, **over):
        kw = dict(lattice=cfg.lattice, dims=cfg.dims, n_species=cfg.n_species, n_shells=cfg.n_shells,
                  epi=cfg.epi(), link_cell=cfg.link_cell, accept=cfg.accept_table(0), seed=cfg.seed)
        kw.update(over)
        return cls(init=init, threads=threads, **kw)

    def set_local_model(self, quad):
        """S12: nonlinear local-energy model; quad = W2[s][a][x][y] (x <= y used), the table given at
        creation is its linear part W1[s][a][x].  None: back to pairwise EPI."""
        if quad is None:
            self._lib.oracle_set_local_model(self._h, None)
            return
        q = np.ascontiguousarray(quad, dtype=np.int32)
        assert q.shape == (self.n_shells, self.n_species, self.n_species, self.n_species)
        self._lib.oracle_set_local_model(self._h, _ptr(q, C.c_int32))

    def site_energy(self, k: int) -> int:
        return int(self._lib.oracle_site_energy(self._h, int(k)))

    def set_threads(self, n: int) -> int:
        """OpenMP threads over the cells of a colour (and over sites in the init / energy / pair-count
        loops); 1 = the plain single-threaded loops.  Results never depend on it (pinned)."""
        self.threads = int(self._lib.oracle_set_threads(self._h, int(n)))
        return self.threads

    def close(self):
        if getattr(self, "_h", None):
            self._lib.oracle_destroy(self._h)
            self._h = None

    __del__ = close

    def init_species(self):
        self._lib.oracle_init_species(self._h)

    def init_composition(self, counts):
        """S10: exactly counts[p] sites of species p, placed by the permutation of S6."""
        c = np.ascontiguousarray(counts, dtype=np.int64)
        assert c.size == self.n_species
        if self._lib.oracle_init_composition(self._h, _ptr(c, C.c_int64)) != 0:
            raise ValueError("counts must be non-negative and sum to n_sites")

    def init_permutation(self, i: int) -> int:
        return int(self._lib.oracle_init_permutation(self._h, C.c_uint64(i)))

    def set_species(self, s):
        s = np.ascontiguousarray(s, dtype=np.uint8)
        assert s.size == self.n_sites
        if self._lib.oracle_set_species(self._h, _ptr(s, C.c_uint8)) != 0:
            raise ValueError("species value out of range")

    def species(self) -> np.ndarray:
        out = np.empty(self.n_sites, dtype=np.uint8)
        self._lib.oracle_get_species(self._h, _ptr(out, C.c_uint8))
        return out

    def set_temperature(self, accept):
        accept = np.ascontiguousarray(accept, dtype=np.uint32)
        self._lib.oracle_set_temperature(self._h, _ptr(accept, C.c_uint32), int(accept.size))

    def energy(self) -> int:
        """H recomputed from scratch (S1)."""
        return int(self._lib.oracle_energy(self._h))

    def running_energy(self) -> int:
        return int(self._lib.oracle_running_energy(self._h))

    def neighbour(self, i: int, s: int, k: int) -> int:
        return int(self._lib.oracle_neighbour(self._h, i, s, k))

    def delta_e(self, i: int, direction: int) -> int:
        return int(self._lib.oracle_delta_e(self._h, i, direction))

    def lc_valid(self) -> bool:
        return bool(self._lib.oracle_lc_valid(self._h))

    def sweep(self, n: int = 1, order_mode: int = 0, order_seed: int = 0):
        if self._lib.oracle_sweep_lc(self._h, int(n), int(order_mode), int(order_seed)) != 0:
            raise ValueError("lattice dimensions not divisible by 2*link_cell")

    def sweep_slabs(self, n: int, n_slabs: int, ghost: int = 2, exchange: bool = True, order_seed: int = 0) -> int:
        """S11: n link-cell sweeps with the lattice cut into n_slabs slabs along z, each holding
        only its window (ghost layers included) and exchanging boundary layers after every colour pass.  Returns
        the number of reads of sites a slab did not hold (0 when the protocol is right)."""
        bad = int(self._lib.oracle_sweep_lc_slabs(self._h, int(n), int(n_slabs), int(ghost), 1 if exchange else 0,
                                                  int(order_seed)))
        if bad < 0:
            raise ValueError("the lattice cannot be cut into that many slabs (pairs of link-cell rows)")
        return bad

    def slab_partition(self, n_slabs: int):
        """[(first link-cell row, number of rows)] of the n_slabs slabs (reading S11)."""
        rows = np.zeros(2 * int(n_slabs), dtype=np.int32)
        if self._lib.oracle_slab_partition(self._h, int(n_slabs), _ptr(rows, C.c_int32)) != 0:
            raise ValueError("the lattice cannot be cut into that many slabs")
        return [(int(rows[2 * k]), int(rows[2 * k + 1])) for k in range(int(n_slabs))]

    def sweep_sequential(self, n: int = 1):
        self._lib.oracle_sweep_seq(self._h, int(n))

    def shift(self, t: int):
        o = np.zeros(3, dtype=np.int32)
        self._lib.oracle_shift(self._h, int(t), _ptr(o, C.c_int32))
        return tuple(int(v) for v in o)

    def stats(self):
        a, b, c = C.c_int64(), C.c_int64(), C.c_int64()
        self._lib.oracle_stats(self._h, C.byref(a), C.byref(b), C.byref(c))
        return a.value, b.value, c.value

    def set_sweep_counter(self, t: int):
        """Resume from a checkpoint: the next sweep is sweep t; the trace restarts there."""
        if self._lib.oracle_set_sweep_counter(self._h, int(t)) != 0:
            raise ValueError("sweep counter out of range")

    def energy_trace(self, first: int = 0, count: int | None = None) -> np.ndarray:
        if count is None:
            count = self.stats()[0] - first
        out = np.zeros(count, dtype=np.int64)
        if self._lib.oracle_trace(self._h, first, count, _ptr(out, C.c_int64)) != count:
            raise IndexError("trace range")
        return out

    def count_visits(self, on: bool = True):
        self._lib.oracle_count_visits(self._h, 1 if on else 0)

    def visits(self) -> np.ndarray:
        out = np.zeros(self.n_sites, dtype=np.uint32)
        self._lib.oracle_get_visits(self._h, _ptr(out, C.c_uint32))
        return out

    def pair_counts(self) -> np.ndarray:
        out = np.zeros((self.n_shells, self.n_species, self.n_species), dtype=np.int64)
        self._lib.oracle_pair_counts(self._h, _ptr(out, C.c_int64))
        return out

    def sro(self):
        """(alpha, pair_counts), both [n_shells][p'][p]; Eq. 8."""
        a = np.zeros((self.n_shells, self.n_species, self.n_species), dtype=np.float64)
        c = np.zeros((self.n_shells, self.n_species, self.n_species), dtype=np.int64)
        self._lib.oracle_sro(self._h, _ptr(a, C.c_double), _ptr(c, C.c_int64))
        return a, c
