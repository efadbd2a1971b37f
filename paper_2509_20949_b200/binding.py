"""ctypes binding for include/smcx.h -- same names, argument marshalling only."""
from __future__ import annotations

import ctypes as C
import os
import re

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.environ.get("SMCX_LIBRARY") or os.path.join(_HERE, "libsmcx.so")  # override: a differently built libsmcx
_HEADER = os.path.join(os.path.dirname(_HERE), "include", "smcx.h")
_lib = None

BCC, FCC = 0, 1
STORAGE_AUTO, STORAGE_2BIT, STORAGE_4BIT, STORAGE_U8 = 0, 2, 4, 8
KERNEL_AUTO, KERNEL_WARP_PER_CELL, KERNEL_THREAD_PER_CELL, KERNEL_THREAD_PERSISTENT, KERNEL_GROUP_PER_CELL = 0, 1, 2, 3, 4
KERNEL_FCC_THREAD = 5
KERNEL_LOCAL_WARP = 6
KERNEL_BCC4_THREAD = 7
MODEL_EPI, MODEL_LOCAL = 0, 1


class SmcxError(RuntimeError):
    def __init__(self, code: int, what: str, detail: str = ""):
        self.code = code
        super().__init__(f"{what}: [{code}] {_strerror(code)}" + (f" ({detail})" if detail else ""))


class _Params(C.Structure):
    _fields_ = [
        ("lattice", C.c_int32), ("dims", C.c_int32 * 3), ("n_species", C.c_int32), ("n_shells", C.c_int32),
        ("epi", C.POINTER(C.c_int32)), ("link_cell", C.c_int32), ("kT_units", C.c_int32),
        ("accept", C.POINTER(C.c_uint32)), ("accept_len", C.c_int32), ("seed", C.c_uint64),
        ("storage", C.c_int32), ("kernel", C.c_int32), ("device", C.c_int32), ("trace_capacity", C.c_int32),
        ("stream", C.c_void_p), ("d_workspace", C.c_void_p), ("workspace_bytes", C.c_size_t),
        ("group_lanes", C.c_int32), ("group_warps", C.c_int32),
        ("domain_count", C.c_int32), ("domain_index", C.c_int32),
        ("model", C.c_int32), ("local_quad", C.POINTER(C.c_int32)),
    ]


class DomainInfo(C.Structure):
    """smcx_domain_info_t"""
    _fields_ = [
        ("n_domains", C.c_int32), ("index", C.c_int32), ("lower", C.c_int32), ("upper", C.c_int32),
        ("row_first", C.c_int32), ("row_count", C.c_int32), ("z_base", C.c_int32), ("z_layers", C.c_int32),
        ("ghost", C.c_int32), ("storage", C.c_int32), ("layer_bytes", C.c_int64), ("owned_sites", C.c_int64),
    ]

    def as_dict(self):
        return {k: int(getattr(self, k)) for k, _ in self._fields_}


class DomainIpc(C.Structure):
    """smcx_domain_ipc_t"""
    _fields_ = [("handle", C.c_ubyte * 64), ("storage_offset", C.c_int64), ("flags_offset", C.c_int64),
                ("index", C.c_int32), ("device", C.c_int32)]

    def to_bytes(self) -> bytes:
        return bytes(self)

    @classmethod
    def from_bytes(cls, b: bytes):
        return cls.from_buffer_copy(b)


class DomainMsg(C.Structure):
    """smcx_domain_msg_t"""
    _fields_ = [("peer", C.c_int32), ("tag", C.c_int32), ("offset", C.c_int64), ("bytes", C.c_int64)]

    def as_tuple(self):
        return (int(self.peer), int(self.tag), int(self.offset), int(self.bytes))


def library_path() -> str:
    return _LIB_PATH


def exported_symbols() -> list:
    """Function names declared in include/smcx.h."""
    text = open(_HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(smcx_[a-z_0-9]+)\s*\(", text)))


def load_library(build_if_missing: bool = True):
    """dlopen libsmcx.so (built in-tree by paper_2509_20949_b200/build.py).  Raises if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if build_if_missing and not os.environ.get("SMCX_LIBRARY"):
        from . import build as _build
        try:
            _build.build()
        except Exception as exc:  # nvcc missing or compile error
            if not os.path.exists(_LIB_PATH):
                raise RuntimeError(f"libsmcx.so is not built and could not be built: {exc}") from exc
    if not os.path.exists(_LIB_PATH):
        raise RuntimeError("libsmcx.so not found; run `python -m paper_2509_20949_b200.build`")
    lib = C.CDLL(_LIB_PATH)
    vp, i64p, i32p = C.c_void_p, C.POINTER(C.c_int64), C.POINTER(C.c_int32)
    sig = {
        "smcx_workspace_bytes": (C.c_int, [C.POINTER(_Params), C.POINTER(C.c_size_t)]),
        "smcx_create": (C.c_int, [C.POINTER(vp), C.POINTER(_Params)]),
        "smcx_destroy": (None, [vp]),
        "smcx_set_species": (C.c_int, [vp, C.POINTER(C.c_uint8)]),
        "smcx_set_species_device": (C.c_int, [vp, vp]),
        "smcx_storage_bytes": (C.c_int, [vp, C.POINTER(C.c_size_t)]),
        "smcx_species_packed": (C.c_int, [vp, vp]),
        "smcx_set_species_packed": (C.c_int, [vp, vp]),
        "smcx_set_temperature": (C.c_int, [vp, C.c_int32, C.POINTER(C.c_uint32), C.c_int32]),
        "smcx_init_composition": (C.c_int, [vp, i64p]),
        "smcx_set_sweep_counter": (C.c_int, [vp, C.c_int64]),
        "smcx_sweep": (C.c_int, [vp, C.c_int64]),
        "smcx_energy": (C.c_int, [vp, i64p]),
        "smcx_running_energy": (C.c_int, [vp, i64p]),
        "smcx_energy_trace": (C.c_int, [vp, C.c_int64, C.c_int64, i64p]),
        "smcx_species": (C.c_int, [vp, C.POINTER(C.c_uint8)]),
        "smcx_species_device": (C.c_int, [vp, vp]),
        "smcx_sro": (C.c_int, [vp, C.POINTER(C.c_double), i64p]),
        "smcx_stats": (C.c_int, [vp, i64p, i64p, i64p]),
        "smcx_synchronize": (C.c_int, [vp]),
        "smcx_shell_offsets": (C.c_int, [vp, C.c_int32, i32p, C.c_int32, i32p]),
        "smcx_get_config": (C.c_int, [vp, i32p, i32p, i64p, i64p]),
        "smcx_kernel_launches": (C.c_int64, [vp]),
        "smcx_pair_counts_static": (C.c_int, [C.c_int32, i32p, C.c_int32, C.c_int32, vp, vp, vp]),
        "smcx_group_layout": (C.c_int, [C.POINTER(_Params), i32p, i32p, i32p, i32p, i32p, i32p, C.POINTER(C.c_uint8)]),
        "smcx_ensemble_create": (C.c_int, [C.POINTER(vp), C.POINTER(_Params), C.c_int32, i32p,
                                           C.POINTER(C.POINTER(C.c_uint32)), i32p, C.POINTER(C.c_uint64), C.c_uint64]),
        "smcx_ensemble_destroy": (None, [vp]),
        "smcx_ensemble_replica": (vp, [vp, C.c_int32]),
        "smcx_ensemble_sweep": (C.c_int, [vp, C.c_int64]),
        "smcx_ensemble_exchange": (C.c_int, [vp, C.c_int32]),
        "smcx_ensemble_run": (C.c_int, [vp, C.c_int64, C.c_int64]),
        "smcx_ensemble_state": (C.c_int, [vp, i32p, i64p, i64p, i64p, i32p, i64p]),
        "smcx_ensemble_synchronize": (C.c_int, [vp]),
        "smcx_ensemble_kernel_launches": (C.c_int64, [vp]),
        "smcx_domain_partition": (C.c_int, [C.POINTER(_Params), C.c_int32, C.c_int32, C.POINTER(DomainInfo)]),
        "smcx_domain_plan_messages": (C.c_int, [C.POINTER(_Params), C.c_int32, C.c_int32, C.c_int64, C.c_int64, C.c_int32,
                                                C.POINTER(DomainMsg), C.POINTER(DomainMsg)]),
        "smcx_domain_workspace_bytes": (C.c_int, [C.POINTER(_Params), C.c_int32, C.c_int32, C.POINTER(C.c_size_t)]),
        "smcx_domain_create": (C.c_int, [C.POINTER(vp), C.POINTER(_Params), C.c_int32, C.c_int32]),
        "smcx_domain_destroy": (None, [vp]),
        "smcx_domain_info": (C.c_int, [vp, C.POINTER(DomainInfo)]),
        "smcx_domain_storage": (vp, [vp]),
        "smcx_domain_set_species": (C.c_int, [vp, C.POINTER(C.c_uint8)]),
        "smcx_domain_species": (C.c_int, [vp, C.POINTER(C.c_uint8)]),
        "smcx_domain_init_composition": (C.c_int, [vp, i64p]),
        "smcx_domain_set_temperature": (C.c_int, [vp, C.c_int32, C.POINTER(C.c_uint32), C.c_int32]),
        "smcx_domain_set_sweep_counter": (C.c_int, [vp, C.c_int64]),
        "smcx_domain_begin_sweep": (C.c_int, [vp, C.POINTER(DomainMsg), C.POINTER(DomainMsg)]),
        "smcx_domain_pass": (C.c_int, [vp, C.c_int32, C.c_int32]),
        "smcx_domain_pass_messages": (C.c_int, [vp, C.c_int32, C.POINTER(DomainMsg), C.POINTER(DomainMsg)]),
        "smcx_domain_end_sweep": (C.c_int, [vp]),
        "smcx_domain_pair_counts": (C.c_int, [vp, i64p]),
        "smcx_domain_running_energy": (C.c_int, [vp, i64p]),
        "smcx_domain_energy_trace": (C.c_int, [vp, C.c_int64, C.c_int64, i64p]),
        "smcx_domain_stats": (C.c_int, [vp, i64p, i64p, i64p]),
        "smcx_domain_synchronize": (C.c_int, [vp]),
        "smcx_domain_kernel_launches": (C.c_int64, [vp]),
        "smcx_sro_from_counts": (C.c_int, [C.POINTER(_Params), i64p, C.POINTER(C.c_double), i64p]),
        "smcx_domain_group_create": (C.c_int, [C.POINTER(vp), C.POINTER(_Params), C.c_int32, i32p, C.c_int32]),
        "smcx_domain_group_destroy": (None, [vp]),
        "smcx_domain_group_member": (vp, [vp, C.c_int32]),
        "smcx_domain_group_sweep": (C.c_int, [vp, C.c_int64]),
        "smcx_domain_group_set_temperature": (C.c_int, [vp, C.c_int32, C.POINTER(C.c_uint32), C.c_int32]),
        "smcx_domain_group_set_species": (C.c_int, [vp, C.POINTER(C.c_uint8)]),
        "smcx_domain_group_init_composition": (C.c_int, [vp, i64p]),
        "smcx_domain_group_set_sweep_counter": (C.c_int, [vp, C.c_int64]),
        "smcx_domain_group_species": (C.c_int, [vp, C.POINTER(C.c_uint8)]),
        "smcx_domain_group_energy": (C.c_int, [vp, i64p]),
        "smcx_domain_group_running_energy": (C.c_int, [vp, i64p]),
        "smcx_domain_group_energy_trace": (C.c_int, [vp, C.c_int64, C.c_int64, i64p]),
        "smcx_domain_group_sro": (C.c_int, [vp, C.POINTER(C.c_double), i64p]),
        "smcx_domain_group_stats": (C.c_int, [vp, i64p, i64p, i64p]),
        "smcx_domain_group_synchronize": (C.c_int, [vp]),
        "smcx_domain_group_kernel_launches": (C.c_int64, [vp]),
        "smcx_domain_group_message_bytes": (C.c_int64, [vp]),
        "smcx_domain_group_fused_messages": (C.c_int64, [vp]),
        "smcx_domain_pass_fused": (C.c_int, [vp, C.c_int32, vp, C.c_int64]),
        "smcx_domain_pass_split": (C.c_int, [vp, C.c_int32, vp]),
        "smcx_domain_ipc_export": (C.c_int, [vp, C.POINTER(DomainIpc)]),
        "smcx_domain_ipc_connect": (C.c_int, [vp, C.POINTER(DomainIpc), C.POINTER(DomainIpc)]),
        "smcx_domain_flags": (vp, [vp]),
        "smcx_domain_connect": (C.c_int, [vp, vp, vp, vp, vp]),
        "smcx_domain_sweep_connected": (C.c_int, [vp, C.c_int64]),
        "smcx_last_error": (C.c_char_p, [vp]),
        "smcx_strerror": (C.c_char_p, [C.c_int]),
        "smcx_version": (C.c_char_p, []),
    }
    for name, (res, args) in sig.items():
        fn = getattr(lib, name)
        fn.restype, fn.argtypes = res, args
    _lib = lib
    return lib


def _strerror(code: int) -> str:
    try:
        return load_library(False).smcx_strerror(code).decode()
    except Exception:
        return "?"


def _make_params(lattice, dims, n_species, n_shells, epi, accept, seed, link_cell, kT_units, storage, kernel,
                 device, trace_capacity, group_lanes=0, group_warps=0, local_quad=None):
    epi = np.ascontiguousarray(epi, dtype=np.int32)
    accept = np.ascontiguousarray(accept, dtype=np.uint32)
    p = _Params()
    p.lattice = int(lattice)
    p.dims = (C.c_int32 * 3)(*[int(d) for d in dims])
    p.n_species, p.n_shells = int(n_species), int(n_shells)
    p.epi = epi.ctypes.data_as(C.POINTER(C.c_int32))
    p.link_cell, p.kT_units = int(link_cell), int(kT_units)
    p.accept = accept.ctypes.data_as(C.POINTER(C.c_uint32))
    p.accept_len = int(accept.size)
    p.seed = int(seed)
    p.storage, p.kernel, p.device, p.trace_capacity = int(storage), int(kernel), int(device), int(trace_capacity)
    p.group_lanes, p.group_warps = int(group_lanes), int(group_warps)
    quad = None
    if local_quad is not None:      # SMCX_MODEL_LOCAL: epi is the linear part W1, local_quad the quadratic part W2
        quad = np.ascontiguousarray(local_quad, dtype=np.int32)
        if quad.shape != (int(n_shells), int(n_species), int(n_species), int(n_species)):
            raise ValueError("local_quad must have shape [n_shells][n_species][n_species][n_species]")
        p.model = MODEL_LOCAL
        p.local_quad = quad.ctypes.data_as(C.POINTER(C.c_int32))
    return p, (epi, accept, quad)


class Lattice:
    """One smcx_t handle.  Methods mirror the C entry points of include/smcx.h."""

    def __init__(self, lattice, dims, n_species, n_shells, epi, accept, seed, link_cell=4, kT_units=0,
                 storage=STORAGE_AUTO, kernel=KERNEL_AUTO, device=0, trace_capacity=0, group_lanes=0, group_warps=0,
                 local_quad=None):
        import torch  # device memory + stream only

        if not torch.cuda.is_available():
            raise RuntimeError("paper_2509_20949_b200 needs a CUDA device; there is no CPU fallback")
        self._lib = lib = load_library()
        self._h = None
        p, keep = _make_params(lattice, dims, n_species, n_shells, epi, accept, seed, link_cell, kT_units, storage,
                               kernel, device, trace_capacity, group_lanes, group_warps, local_quad)
        need = C.c_size_t(0)
        rc = lib.smcx_workspace_bytes(C.byref(p), C.byref(need))
        if rc != 0:
            raise SmcxError(rc, "smcx_workspace_bytes")
        self.device = torch.device("cuda", int(device))
        with torch.cuda.device(self.device):
            self._workspace = torch.empty(int(need.value), dtype=torch.uint8, device=self.device)
            self._stream = torch.cuda.current_stream(self.device)
        p.stream = C.c_void_p(self._stream.cuda_stream)
        p.d_workspace = C.c_void_p(self._workspace.data_ptr())
        p.workspace_bytes = int(need.value)
        h = C.c_void_p()
        rc = lib.smcx_create(C.byref(h), C.byref(p))
        if rc != 0:
            raise SmcxError(rc, "smcx_create")
        self._h = h
        del keep
        self.lattice, self.dims = int(lattice), tuple(int(d) for d in dims)
        self.n_species, self.n_shells = int(n_species), int(n_shells)
        st, kn, ns, nc = C.c_int32(), C.c_int32(), C.c_int64(), C.c_int64()
        self._check(lib.smcx_get_config(h, C.byref(st), C.byref(kn), C.byref(ns), C.byref(nc)), "smcx_get_config")
        self.storage, self.kernel, self.n_sites, self.n_cells = st.value, kn.value, ns.value, nc.value

    @classmethod
    def _borrowed(cls, handle, owner, lattice, dims, n_species, n_shells, device):
        """Wrap a handle owned by an Ensemble (smcx_ensemble_replica): never destroyed from here."""
        import torch
        self = cls.__new__(cls)
        self._lib = load_library()
        self._h = C.c_void_p(handle)
        self._owner, self._borrowed_handle = owner, True
        self._workspace = None
        self.device = torch.device("cuda", int(device))
        self.lattice, self.dims = int(lattice), tuple(int(d) for d in dims)
        self.n_species, self.n_shells = int(n_species), int(n_shells)
        st, kn, ns, nc = C.c_int32(), C.c_int32(), C.c_int64(), C.c_int64()
        self._check(self._lib.smcx_get_config(self._h, C.byref(st), C.byref(kn), C.byref(ns), C.byref(nc)), "smcx_get_config")
        self.storage, self.kernel, self.n_sites, self.n_cells = st.value, kn.value, ns.value, nc.value
        return self

    @classmethod
    def from_config(cls, cfg, **over):
        kw = dict(lattice=cfg.lattice, dims=cfg.dims, n_species=cfg.n_species, n_shells=cfg.n_shells, epi=cfg.epi(),
                  accept=cfg.accept_table(0), seed=cfg.seed, link_cell=cfg.link_cell, kT_units=cfg.kT_at(0))
        kw.update(over)
        return cls(**kw)

    # -- plumbing ---------------------------------------------------------------------------
    def _check(self, rc, what):
        if rc != 0:
            detail = self._lib.smcx_last_error(self._h).decode() if self._h else ""
            raise SmcxError(rc, what, detail)

    def close(self):
        if getattr(self, "_borrowed_handle", False):
            self._h = None
            return
        if getattr(self, "_h", None):
            self._lib.smcx_destroy(self._h)
            self._h = None
            self._workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- smcx.h -----------------------------------------------------------------------------
    def set_species(self, species):
        s = np.ascontiguousarray(species, dtype=np.uint8)
        if s.size != self.n_sites:
            raise ValueError("species must have n_sites entries")
        self._check(self._lib.smcx_set_species(self._h, s.ctypes.data_as(C.POINTER(C.c_uint8))), "smcx_set_species")

    def set_species_device(self, tensor):
        assert tensor.is_cuda and tensor.dtype.itemsize == 1 and tensor.numel() == self.n_sites and tensor.is_contiguous()
        self._check(self._lib.smcx_set_species_device(self._h, C.c_void_p(tensor.data_ptr())), "smcx_set_species_device")

    def storage_bytes(self) -> int:
        n = C.c_size_t(0)
        self._check(self._lib.smcx_storage_bytes(self._h, C.byref(n)), "smcx_storage_bytes")
        return int(n.value)

    def species_packed(self, out=None) -> np.ndarray:
        """The species array in device storage format (smcx_species_packed), as bytes."""
        n = self.storage_bytes()
        if out is None:
            out = np.empty(n, dtype=np.uint8)
        assert out.dtype == np.uint8 and out.size == n and out.flags.c_contiguous
        self._check(self._lib.smcx_species_packed(self._h, C.c_void_p(out.ctypes.data)), "smcx_species_packed")
        return out

    def set_species_packed(self, packed):
        a = np.ascontiguousarray(packed, dtype=np.uint8)
        if a.size != self.storage_bytes():
            raise ValueError("packed array must have storage_bytes() bytes")
        self._check(self._lib.smcx_set_species_packed(self._h, C.c_void_p(a.ctypes.data)), "smcx_set_species_packed")

    def init_composition(self, counts):
        c = np.ascontiguousarray(counts, dtype=np.int64)
        if c.size != self.n_species:
            raise ValueError("counts must have n_species entries")
        self._check(self._lib.smcx_init_composition(self._h, c.ctypes.data_as(C.POINTER(C.c_int64))), "smcx_init_composition")

    def set_sweep_counter(self, t):
        self._check(self._lib.smcx_set_sweep_counter(self._h, int(t)), "smcx_set_sweep_counter")

    def set_temperature(self, kT_units, accept):
        a = np.ascontiguousarray(accept, dtype=np.uint32)
        self._check(self._lib.smcx_set_temperature(self._h, int(kT_units), a.ctypes.data_as(C.POINTER(C.c_uint32)),
                                                   int(a.size)), "smcx_set_temperature")

    def sweep(self, n=1):
        self._check(self._lib.smcx_sweep(self._h, int(n)), "smcx_sweep")

    def energy(self) -> int:
        e = C.c_int64()
        self._check(self._lib.smcx_energy(self._h, C.byref(e)), "smcx_energy")
        return e.value

    def running_energy(self) -> int:
        e = C.c_int64()
        self._check(self._lib.smcx_running_energy(self._h, C.byref(e)), "smcx_running_energy")
        return e.value

    def energy_trace(self, first=0, count=None) -> np.ndarray:
        if count is None:
            count = self.stats()[0] - first
        out = np.zeros(int(count), dtype=np.int64)
        self._check(self._lib.smcx_energy_trace(self._h, int(first), int(count), out.ctypes.data_as(C.POINTER(C.c_int64))),
                    "smcx_energy_trace")
        return out

    def species(self, out=None) -> np.ndarray:
        if out is None:
            out = np.empty(self.n_sites, dtype=np.uint8)
        assert out.dtype == np.uint8 and out.size == self.n_sites and out.flags.c_contiguous
        self._check(self._lib.smcx_species(self._h, out.ctypes.data_as(C.POINTER(C.c_uint8))), "smcx_species")
        return out

    def species_device(self, out=None):
        import torch
        if out is None:
            out = torch.empty(self.n_sites, dtype=torch.uint8, device=self.device)
        self._check(self._lib.smcx_species_device(self._h, C.c_void_p(out.data_ptr())), "smcx_species_device")
        return out

    def sro(self):
        shape = (self.n_shells, self.n_species, self.n_species)
        alpha = np.zeros(shape, dtype=np.float64)
        counts = np.zeros(shape, dtype=np.int64)
        self._check(self._lib.smcx_sro(self._h, alpha.ctypes.data_as(C.POINTER(C.c_double)),
                                       counts.ctypes.data_as(C.POINTER(C.c_int64))), "smcx_sro")
        return alpha, counts

    def stats(self):
        a, b, c = C.c_int64(), C.c_int64(), C.c_int64()
        self._check(self._lib.smcx_stats(self._h, C.byref(a), C.byref(b), C.byref(c)), "smcx_stats")
        return a.value, b.value, c.value

    def synchronize(self):
        self._check(self._lib.smcx_synchronize(self._h), "smcx_synchronize")

    def shell_offsets(self, shell) -> np.ndarray:
        buf = np.zeros((64, 3), dtype=np.int32)
        n = C.c_int32()
        self._check(self._lib.smcx_shell_offsets(self._h, int(shell), buf.ctypes.data_as(C.POINTER(C.c_int32)), 64,
                                                 C.byref(n)), "smcx_shell_offsets")
        return buf[: n.value].copy()

    @property
    def kernel_launches(self) -> int:
        return int(self._lib.smcx_kernel_launches(self._h))


class Ensemble:
    """One smcx_ensemble_t: replicas of one system on a temperature ladder with replica exchange on
    the device (include/smcx.h, "Temperature parallelism on one GPU").  Methods mirror the C calls."""

    def __init__(self, lattice, dims, n_species, n_shells, epi, kT_units, accept_tables, seeds, exchange_seed,
                 link_cell=4, storage=STORAGE_AUTO, kernel=KERNEL_AUTO, device=0, trace_capacity=0):
        import torch

        if not torch.cuda.is_available():
            raise RuntimeError("paper_2509_20949_b200 needs a CUDA device; there is no CPU fallback")
        self._lib = lib = load_library()
        self._e = None
        n = len(kT_units)
        if not (len(accept_tables) == n and len(seeds) == n):
            raise ValueError("kT_units, accept_tables and seeds must have one entry per replica")
        tabs = [np.ascontiguousarray(t, dtype=np.uint32) for t in accept_tables]
        p, keep = _make_params(lattice, dims, n_species, n_shells, epi, tabs[0], 0, link_cell, 0, storage, kernel,
                               device, trace_capacity)
        self.device = torch.device("cuda", int(device))
        with torch.cuda.device(self.device):
            self._stream = torch.cuda.current_stream(self.device)
        p.stream = C.c_void_p(self._stream.cuda_stream)
        kT = (C.c_int32 * n)(*[int(k) for k in kT_units])
        ptrs = (C.POINTER(C.c_uint32) * n)(*[t.ctypes.data_as(C.POINTER(C.c_uint32)) for t in tabs])
        lens = (C.c_int32 * n)(*[int(t.size) for t in tabs])
        sd = (C.c_uint64 * n)(*[int(s) for s in seeds])
        e = C.c_void_p()
        rc = lib.smcx_ensemble_create(C.byref(e), C.byref(p), n, kT, ptrs, lens, sd, C.c_uint64(int(exchange_seed)))
        if rc != 0:
            raise SmcxError(rc, "smcx_ensemble_create")
        self._e = e
        del keep
        self.n_replicas = n
        self.kT_units = [int(k) for k in kT_units]
        self.replicas = [Lattice._borrowed(lib.smcx_ensemble_replica(e, r), self, lattice, dims, n_species, n_shells,
                                           device) for r in range(n)]

    def _check(self, rc, what):
        if rc != 0:
            raise SmcxError(rc, what)

    def close(self):
        if getattr(self, "_e", None):
            for r in self.replicas:
                r.close()
            self._lib.smcx_ensemble_destroy(self._e)
            self._e = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def sweep(self, n=1):
        self._check(self._lib.smcx_ensemble_sweep(self._e, int(n)), "smcx_ensemble_sweep")

    def exchange(self, parity):
        self._check(self._lib.smcx_ensemble_exchange(self._e, int(parity)), "smcx_ensemble_exchange")

    def run(self, rounds, sweeps_per_round):
        self._check(self._lib.smcx_ensemble_run(self._e, int(rounds), int(sweeps_per_round)), "smcx_ensemble_run")

    def synchronize(self):
        self._check(self._lib.smcx_ensemble_synchronize(self._e), "smcx_ensemble_synchronize")

    def state(self) -> dict:
        n = self.n_replicas
        ras = np.zeros(n, dtype=np.int32)
        en = np.zeros(n, dtype=np.int64)
        att, acc = np.zeros(n - 1, dtype=np.int64), np.zeros(n - 1, dtype=np.int64)
        flg = np.zeros(n - 1, dtype=np.int32)
        rounds = C.c_int64()
        i32p, i64p = C.POINTER(C.c_int32), C.POINTER(C.c_int64)
        self._check(self._lib.smcx_ensemble_state(self._e, ras.ctypes.data_as(i32p), en.ctypes.data_as(i64p),
                                                  att.ctypes.data_as(i64p), acc.ctypes.data_as(i64p),
                                                  flg.ctypes.data_as(i32p), C.byref(rounds)), "smcx_ensemble_state")
        return dict(replica_at_slot=ras, energy_at_slot=en, attempted=att, accepted=acc, last_flags=flg,
                    rounds=rounds.value)

    @property
    def kernel_launches(self) -> int:
        return int(self._lib.smcx_ensemble_kernel_launches(self._e))


def group_layout(**kw) -> dict:
    """smcx_group_layout: the tile layout the host picks for the sub-warp kernel (no GPU needed)."""
    lib = load_library()
    defaults = dict(link_cell=4, kT_units=0, storage=0, kernel=0, device=0, trace_capacity=0)
    defaults.update(kw)
    p, _keep = _make_params(**defaults)
    v = [C.c_int32() for _ in range(6)]
    slots = (C.c_uint8 * 128)()
    rc = lib.smcx_group_layout(C.byref(p), *[C.byref(x) for x in v], slots)
    if rc != 0:
        raise SmcxError(rc, "smcx_group_layout")
    names = ("lanes", "A", "B", "shift", "tile_bytes", "skew")
    out = {k: x.value for k, x in zip(names, v)}
    out["slots"] = np.frombuffer(bytes(slots), dtype=np.uint8).copy()
    return out


def workspace_bytes(**kw) -> int:
    lib = load_library()
    defaults = dict(link_cell=4, kT_units=0, storage=0, kernel=0, device=0, trace_capacity=0)
    defaults.update(kw)
    p, _keep = _make_params(**defaults)
    need = C.c_size_t(0)
    rc = lib.smcx_workspace_bytes(C.byref(p), C.byref(need))
    if rc != 0:
        raise SmcxError(rc, "smcx_workspace_bytes")
    return int(need.value)


# ---- lattice parallelism (include/smcx.h, "Lattice parallelism: slabs with ghost layers") -----------------------
def domain_partition(n_domains, index, **kw) -> dict:
    """smcx_domain_partition: what slab `index` of `n_domains` holds (host arithmetic, no GPU needed)."""
    lib = load_library()
    defaults = dict(link_cell=4, kT_units=0, storage=0, kernel=0, device=0, trace_capacity=0)
    defaults.update(kw)
    p, _keep = _make_params(**defaults)
    info = DomainInfo()
    rc = lib.smcx_domain_partition(C.byref(p), int(n_domains), int(index), C.byref(info))
    if rc != 0:
        raise SmcxError(rc, "smcx_domain_partition")
    return info.as_dict()


def domain_plan_messages(n_domains, index, sweep, phase, first_sweep=0, **kw):
    """smcx_domain_plan_messages: (send, recv), each (peer, tag, offset, bytes), of a slab in one phase
    (-1 = window shift at the start of the sweep, 0..7 = after that colour pass).  Host arithmetic, no GPU needed."""
    lib = load_library()
    defaults = dict(link_cell=4, kT_units=0, storage=0, kernel=0, device=0, trace_capacity=0)
    defaults.update(kw)
    p, _keep = _make_params(**defaults)
    send, recv = DomainMsg(), DomainMsg()
    rc = lib.smcx_domain_plan_messages(C.byref(p), int(n_domains), int(index), int(sweep), int(first_sweep), int(phase),
                                       C.byref(send), C.byref(recv))
    if rc != 0:
        raise SmcxError(rc, "smcx_domain_plan_messages")
    return send.as_tuple(), recv.as_tuple()


STATIC_PAIR_COUNTS_MAX = 1024


def pair_counts_static(lattice, dims, n_species, n_shells, d_species, d_pair_counts, stream=None):
    """smcx_pair_counts_static: ordered pair counts of the uint8 device tensor `d_species` into the int64 device tensor
    `d_pair_counts` ([n_shells][n_species][n_species]) with the library's static device scratch: no device allocation,
    no handle, no synchronisation.  Both tensors are the caller's."""
    lib = load_library()
    d = (C.c_int32 * 3)(*[int(x) for x in dims])
    sp = int(stream.cuda_stream) if stream is not None else 0
    rc = lib.smcx_pair_counts_static(int(lattice), d, int(n_species), int(n_shells), C.c_void_p(d_species.data_ptr()),
                                     C.c_void_p(d_pair_counts.data_ptr()), C.c_void_p(sp))
    if rc != 0:
        raise SmcxError(rc, "smcx_pair_counts_static")
    return d_pair_counts


def sro_from_counts(half_counts, **kw):
    """smcx_sro_from_counts: (alpha, ordered pair counts) of the whole lattice from the summed positive-half counts."""
    lib = load_library()
    defaults = dict(link_cell=4, kT_units=0, storage=0, kernel=0, device=0, trace_capacity=0)
    defaults.update(kw)
    p, _keep = _make_params(**defaults)
    shape = (int(p.n_shells), int(p.n_species), int(p.n_species))
    m = np.ascontiguousarray(half_counts, dtype=np.int64).reshape(shape)
    alpha = np.zeros(shape, dtype=np.float64)
    counts = np.zeros(shape, dtype=np.int64)
    rc = lib.smcx_sro_from_counts(C.byref(p), m.ctypes.data_as(C.POINTER(C.c_int64)), alpha.ctypes.data_as(C.POINTER(C.c_double)),
                                  counts.ctypes.data_as(C.POINTER(C.c_int64)))
    if rc != 0:
        raise SmcxError(rc, "smcx_sro_from_counts")
    return alpha, counts


class Domain:
    """One smcx_domain_t: slab `index` of a lattice cut into `n_domains` slabs along z.  The workspace is a torch
    uint8 tensor, so a caller can hand slices of the species storage (`storage_view`) to torch.distributed."""

    def __init__(self, n_domains, index, lattice, dims, n_species, n_shells, epi, accept, seed, link_cell=4, kT_units=0,
                 storage=STORAGE_AUTO, kernel=KERNEL_AUTO, device=0, trace_capacity=0, stream=None, local_quad=None,
                 library_workspace=False):
        import torch

        if not torch.cuda.is_available():
            raise RuntimeError("paper_2509_20949_b200 needs a CUDA device; there is no CPU fallback")
        self._lib = lib = load_library()
        self._d = None
        p, keep = _make_params(lattice, dims, n_species, n_shells, epi, accept, seed, link_cell, kT_units, storage,
                               kernel, device, trace_capacity, local_quad=local_quad)
        need = C.c_size_t(0)
        rc = lib.smcx_domain_workspace_bytes(C.byref(p), int(n_domains), int(index), C.byref(need))
        if rc != 0:
            raise SmcxError(rc, "smcx_domain_workspace_bytes")
        self.device = torch.device("cuda", int(device))
        with torch.cuda.device(self.device):
            # library_workspace: the library allocates (cudaMalloc), which smcx_domain_ipc_export needs; else a torch tensor
            self._workspace = None if library_workspace else torch.empty(int(need.value), dtype=torch.uint8, device=self.device)
            self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        p.stream = C.c_void_p(self._stream.cuda_stream)
        if self._workspace is not None:
            p.d_workspace = C.c_void_p(self._workspace.data_ptr())
            p.workspace_bytes = int(need.value)
        d = C.c_void_p()
        rc = lib.smcx_domain_create(C.byref(d), C.byref(p), int(n_domains), int(index))
        if rc != 0:
            raise SmcxError(rc, "smcx_domain_create")
        self._d = d
        del keep
        info = DomainInfo()
        self._check(lib.smcx_domain_info(d, C.byref(info)), "smcx_domain_info")
        self.info = info.as_dict()
        self.n_domains, self.index = int(n_domains), int(index)
        self.n_species, self.n_shells = int(n_species), int(n_shells)
        self.n_sites_whole = int(np.prod([int(x) for x in dims])) * (2 if int(lattice) == BCC else 4)
        self._storage_view = None
        if self._workspace is not None:
            off = int(lib.smcx_domain_storage(d)) - self._workspace.data_ptr()
            self._storage_view = self._workspace[off: off + self.info["z_layers"] * self.info["layer_bytes"]]

    @classmethod
    def _borrowed(cls, handle, owner, n_species, n_shells, n_sites_whole):
        self = cls.__new__(cls)
        self._lib = load_library()
        self._d = C.c_void_p(handle)
        self._owner, self._borrowed_handle = owner, True
        self._workspace = self._storage_view = None
        info = DomainInfo()
        self._check(self._lib.smcx_domain_info(self._d, C.byref(info)), "smcx_domain_info")
        self.info = info.as_dict()
        self.n_domains, self.index = self.info["n_domains"], self.info["index"]
        self.n_species, self.n_shells, self.n_sites_whole = int(n_species), int(n_shells), int(n_sites_whole)
        return self

    def _check(self, rc, what):
        if rc != 0:
            raise SmcxError(rc, what)

    def close(self):
        if getattr(self, "_borrowed_handle", False):
            self._d = None
            return
        if getattr(self, "_d", None):
            self._lib.smcx_domain_destroy(self._d)
            self._d = None
            self._workspace = self._storage_view = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def storage_view(self, msg):
        """The bytes of message (peer, tag, offset, bytes) as a view of the workspace tensor."""
        _, _, off, n = msg
        return self._storage_view[off: off + n]

    def set_species(self, whole):
        s = np.ascontiguousarray(whole, dtype=np.uint8)
        if s.size != self.n_sites_whole:
            raise ValueError("the array must hold the whole lattice")
        self._check(self._lib.smcx_domain_set_species(self._d, s.ctypes.data_as(C.POINTER(C.c_uint8))), "smcx_domain_set_species")

    def species_into(self, whole):
        """Write the layers this slab owns into `whole` (uint8 array of the whole lattice)."""
        assert whole.dtype == np.uint8 and whole.size == self.n_sites_whole and whole.flags.c_contiguous
        self._check(self._lib.smcx_domain_species(self._d, whole.ctypes.data_as(C.POINTER(C.c_uint8))), "smcx_domain_species")
        return whole

    def init_composition(self, counts):
        c = np.ascontiguousarray(counts, dtype=np.int64)
        self._check(self._lib.smcx_domain_init_composition(self._d, c.ctypes.data_as(C.POINTER(C.c_int64))), "smcx_domain_init_composition")

    def set_temperature(self, kT_units, accept):
        a = np.ascontiguousarray(accept, dtype=np.uint32)
        self._check(self._lib.smcx_domain_set_temperature(self._d, int(kT_units), a.ctypes.data_as(C.POINTER(C.c_uint32)),
                                                          int(a.size)), "smcx_domain_set_temperature")

    def set_sweep_counter(self, t):
        self._check(self._lib.smcx_domain_set_sweep_counter(self._d, int(t)), "smcx_domain_set_sweep_counter")

    def begin_sweep(self):
        send, recv = DomainMsg(), DomainMsg()
        self._check(self._lib.smcx_domain_begin_sweep(self._d, C.byref(send), C.byref(recv)), "smcx_domain_begin_sweep")
        return send.as_tuple(), recv.as_tuple()

    def run_pass(self, colour, part=0):
        self._check(self._lib.smcx_domain_pass(self._d, int(colour), int(part)), "smcx_domain_pass")

    # -- connected slabs: one slab per process, no host in the data path ---------------------------------------------
    def ipc_export(self) -> bytes:
        """smcx_domain_ipc_export as bytes (to hand to the neighbours' processes)."""
        out = DomainIpc()
        self._check(self._lib.smcx_domain_ipc_export(self._d, C.byref(out)), "smcx_domain_ipc_export")
        return out.to_bytes()

    def ipc_connect(self, lower: bytes, upper: bytes):
        lo, up = DomainIpc.from_bytes(lower), DomainIpc.from_bytes(upper)
        self._check(self._lib.smcx_domain_ipc_connect(self._d, C.byref(lo), C.byref(up)), "smcx_domain_ipc_connect")

    @property
    def flags_ptr(self) -> int:
        return int(self._lib.smcx_domain_flags(self._d))

    def connect(self, lower, upper):
        """smcx_domain_connect with neighbours that live in this process (Domain objects)."""
        self._check(self._lib.smcx_domain_connect(self._d, C.c_void_p(lower.storage_ptr), C.c_void_p(lower.flags_ptr),
                                                  C.c_void_p(upper.storage_ptr), C.c_void_p(upper.flags_ptr)), "smcx_domain_connect")

    def sweep_connected(self, n=1):
        self._check(self._lib.smcx_domain_sweep_connected(self._d, int(n)), "smcx_domain_sweep_connected")

    def run_pass_split(self, colour, side_stream):
        """smcx_domain_pass_split: boundary row on `side_stream` (a torch.cuda.Stream), the other rows on the slab's stream."""
        self._check(self._lib.smcx_domain_pass_split(self._d, int(colour), C.c_void_p(side_stream.cuda_stream)), "smcx_domain_pass_split")

    def run_pass_fused(self, colour, peer_storage_ptr, peer_offset):
        """smcx_domain_pass_fused: the boundary row of the pass, storing its message into the neighbour's storage."""
        self._check(self._lib.smcx_domain_pass_fused(self._d, int(colour), C.c_void_p(int(peer_storage_ptr)), int(peer_offset)),
                    "smcx_domain_pass_fused")

    @property
    def storage_ptr(self) -> int:
        return int(self._lib.smcx_domain_storage(self._d))

    def pass_messages(self, colour):
        send, recv = DomainMsg(), DomainMsg()
        self._check(self._lib.smcx_domain_pass_messages(self._d, int(colour), C.byref(send), C.byref(recv)), "smcx_domain_pass_messages")
        return send.as_tuple(), recv.as_tuple()

    def end_sweep(self):
        self._check(self._lib.smcx_domain_end_sweep(self._d), "smcx_domain_end_sweep")

    def pair_counts(self) -> np.ndarray:
        m = np.zeros((self.n_shells, self.n_species, self.n_species), dtype=np.int64)
        self._check(self._lib.smcx_domain_pair_counts(self._d, m.ctypes.data_as(C.POINTER(C.c_int64))), "smcx_domain_pair_counts")
        return m

    def running_energy(self) -> int:
        e = C.c_int64()
        self._check(self._lib.smcx_domain_running_energy(self._d, C.byref(e)), "smcx_domain_running_energy")
        return e.value

    def energy_trace(self, first=0, count=None) -> np.ndarray:
        if count is None:
            count = self.stats()[0] - first
        out = np.zeros(int(count), dtype=np.int64)
        self._check(self._lib.smcx_domain_energy_trace(self._d, int(first), int(count), out.ctypes.data_as(C.POINTER(C.c_int64))),
                    "smcx_domain_energy_trace")
        return out

    def stats(self):
        a, b, c = C.c_int64(), C.c_int64(), C.c_int64()
        self._check(self._lib.smcx_domain_stats(self._d, C.byref(a), C.byref(b), C.byref(c)), "smcx_domain_stats")
        return a.value, b.value, c.value

    def synchronize(self):
        self._check(self._lib.smcx_domain_synchronize(self._d), "smcx_domain_synchronize")

    @property
    def kernel_launches(self) -> int:
        return int(self._lib.smcx_domain_kernel_launches(self._d))


class DomainGroup:
    """One smcx_domain_group_t: every slab of a lattice in this process (on one device or several), messages moved by
    device-to-device / peer copies.  Same results as a Lattice of the whole."""

    def __init__(self, n_domains, lattice, dims, n_species, n_shells, epi, accept, seed, link_cell=4, kT_units=0,
                 storage=STORAGE_AUTO, kernel=KERNEL_AUTO, device=0, devices=None, overlap=True, trace_capacity=0,
                 local_quad=None):
        import torch

        if not torch.cuda.is_available():
            raise RuntimeError("paper_2509_20949_b200 needs a CUDA device; there is no CPU fallback")
        self._lib = lib = load_library()
        self._g = None
        p, keep = _make_params(lattice, dims, n_species, n_shells, epi, accept, seed, link_cell, kT_units, storage,
                               kernel, device, trace_capacity, local_quad=local_quad)
        self.device = torch.device("cuda", int(device))
        with torch.cuda.device(self.device):
            self._stream = torch.cuda.current_stream(self.device)
        p.stream = C.c_void_p(self._stream.cuda_stream)
        dev = None
        if devices is not None:
            if len(devices) != n_domains:
                raise ValueError("devices must have one entry per slab")
            dev = (C.c_int32 * n_domains)(*[int(x) for x in devices])
        g = C.c_void_p()
        rc = lib.smcx_domain_group_create(C.byref(g), C.byref(p), int(n_domains), dev, int(overlap))   # 0 / 1 (True) / 2
        if rc != 0:
            raise SmcxError(rc, "smcx_domain_group_create")
        self._g = g
        del keep
        self.n_domains = int(n_domains)
        self.lattice, self.dims = int(lattice), tuple(int(d) for d in dims)
        self.n_species, self.n_shells = int(n_species), int(n_shells)
        self.n_sites = int(np.prod(self.dims)) * (2 if self.lattice == BCC else 4)
        self.members = [Domain._borrowed(lib.smcx_domain_group_member(g, k), self, n_species, n_shells, self.n_sites)
                        for k in range(self.n_domains)]

    @classmethod
    def from_config(cls, cfg, n_domains, **over):
        kw = dict(lattice=cfg.lattice, dims=cfg.dims, n_species=cfg.n_species, n_shells=cfg.n_shells, epi=cfg.epi(),
                  accept=cfg.accept_table(0), seed=cfg.seed, link_cell=cfg.link_cell, kT_units=cfg.kT_at(0))
        kw.update(over)
        return cls(n_domains, **kw)

    def _check(self, rc, what):
        if rc != 0:
            raise SmcxError(rc, what)

    def close(self):
        if getattr(self, "_g", None):
            for m in self.members:
                m.close()
            self._lib.smcx_domain_group_destroy(self._g)
            self._g = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def sweep(self, n=1):
        self._check(self._lib.smcx_domain_group_sweep(self._g, int(n)), "smcx_domain_group_sweep")

    def set_temperature(self, kT_units, accept):
        a = np.ascontiguousarray(accept, dtype=np.uint32)
        self._check(self._lib.smcx_domain_group_set_temperature(self._g, int(kT_units), a.ctypes.data_as(C.POINTER(C.c_uint32)),
                                                                int(a.size)), "smcx_domain_group_set_temperature")

    def set_species(self, species):
        s = np.ascontiguousarray(species, dtype=np.uint8)
        if s.size != self.n_sites:
            raise ValueError("species must have n_sites entries")
        self._check(self._lib.smcx_domain_group_set_species(self._g, s.ctypes.data_as(C.POINTER(C.c_uint8))), "smcx_domain_group_set_species")

    def init_composition(self, counts):
        c = np.ascontiguousarray(counts, dtype=np.int64)
        self._check(self._lib.smcx_domain_group_init_composition(self._g, c.ctypes.data_as(C.POINTER(C.c_int64))),
                    "smcx_domain_group_init_composition")

    def set_sweep_counter(self, t):
        self._check(self._lib.smcx_domain_group_set_sweep_counter(self._g, int(t)), "smcx_domain_group_set_sweep_counter")

    def species(self, out=None) -> np.ndarray:
        if out is None:
            out = np.empty(self.n_sites, dtype=np.uint8)
        assert out.dtype == np.uint8 and out.size == self.n_sites and out.flags.c_contiguous
        self._check(self._lib.smcx_domain_group_species(self._g, out.ctypes.data_as(C.POINTER(C.c_uint8))), "smcx_domain_group_species")
        return out

    def energy(self) -> int:
        e = C.c_int64()
        self._check(self._lib.smcx_domain_group_energy(self._g, C.byref(e)), "smcx_domain_group_energy")
        return e.value

    def running_energy(self) -> int:
        e = C.c_int64()
        self._check(self._lib.smcx_domain_group_running_energy(self._g, C.byref(e)), "smcx_domain_group_running_energy")
        return e.value

    def energy_trace(self, first=0, count=None) -> np.ndarray:
        if count is None:
            count = self.stats()[0] - first
        out = np.zeros(int(count), dtype=np.int64)
        self._check(self._lib.smcx_domain_group_energy_trace(self._g, int(first), int(count),
                                                             out.ctypes.data_as(C.POINTER(C.c_int64))), "smcx_domain_group_energy_trace")
        return out

    def sro(self):
        shape = (self.n_shells, self.n_species, self.n_species)
        alpha = np.zeros(shape, dtype=np.float64)
        counts = np.zeros(shape, dtype=np.int64)
        self._check(self._lib.smcx_domain_group_sro(self._g, alpha.ctypes.data_as(C.POINTER(C.c_double)),
                                                    counts.ctypes.data_as(C.POINTER(C.c_int64))), "smcx_domain_group_sro")
        return alpha, counts

    def stats(self):
        a, b, c = C.c_int64(), C.c_int64(), C.c_int64()
        self._check(self._lib.smcx_domain_group_stats(self._g, C.byref(a), C.byref(b), C.byref(c)), "smcx_domain_group_stats")
        return a.value, b.value, c.value

    def synchronize(self):
        self._check(self._lib.smcx_domain_group_synchronize(self._g), "smcx_domain_group_synchronize")

    @property
    def kernel_launches(self) -> int:
        return int(self._lib.smcx_domain_group_kernel_launches(self._g))

    @property
    def message_bytes(self) -> int:
        return int(self._lib.smcx_domain_group_message_bytes(self._g))

    @property
    def fused_messages(self) -> int:
        return int(self._lib.smcx_domain_group_fused_messages(self._g))
