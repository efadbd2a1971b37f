"""Host-side checks of the C-ABI library that need no GPU: it loads, exports every symbol that
include/smcx.h declares, and validates parameters with the documented error codes."""
import ctypes as C

import numpy as np
import pytest

import paper_2509_20949_b200 as smcx
from paper_2509_20949_b200.binding import SmcxError, workspace_bytes
from smcx_inputs import get_config, make_accept_table, make_epi

E = dict(NULL_ARG=-1, BAD_LATTICE=-2, BAD_DIMS=-3, BAD_SPECIES=-4, BAD_SHELLS=-5, EPI_NOT_SYMMETRIC=-6,
         LINK_CELL_TOO_SMALL=-7, BAD_TABLE=-8, UNSUPPORTED=-12, EPI_RANGE=-14)


def test_library_loads_and_exports_every_declared_symbol():
    lib = smcx.load_library()
    names = smcx.exported_symbols()
    assert len(names) >= 20 and "smcx_create" in names and "smcx_sweep" in names and "smcx_sro" in names
    for name in names:
        assert hasattr(lib, name), name
    assert b"sm_100a" in lib.smcx_version()
    assert lib.smcx_strerror(0) == b"ok" and lib.smcx_strerror(-3) != lib.smcx_strerror(-4)


def _kw(**over):
    kw = dict(lattice=0, dims=(16, 16, 16), n_species=4, n_shells=2, epi=make_epi(2, 4, 300, 1),
              accept=make_accept_table(600), seed=1, link_cell=4)
    kw.update(over)
    return kw


def _code(**over):
    with pytest.raises(SmcxError) as ei:
        workspace_bytes(**_kw(**over))
    return ei.value.code


def test_workspace_size_covers_the_species_array():
    for k in (1, 2, 3, 4, 5):
        c = get_config(k)
        for storage, per_site in ((smcx.STORAGE_U8, 1.0), (smcx.STORAGE_2BIT, 0.25)):
            if storage == smcx.STORAGE_2BIT:
                continue  # thread-per-cell path is validated separately
            need = workspace_bytes(lattice=c.lattice, dims=c.dims, n_species=c.n_species, n_shells=c.n_shells,
                                   epi=c.epi(), accept=c.accept_table(), seed=c.seed, storage=storage)
            assert c.n_sites * per_site <= need <= c.n_sites * per_site + (16 << 20)


def test_parameter_validation_codes():
    assert _code(lattice=2) == E["BAD_LATTICE"]
    assert _code(dims=(16, 16, 12)) == E["BAD_DIMS"]          # not divisible by 2w
    assert _code(dims=(0, 16, 16)) == E["BAD_DIMS"]
    assert _code(dims=(4, 4, 4), link_cell=2) == E["BAD_DIMS"]  # smaller than a cell plus its halo
    assert _code(n_species=1, epi=np.zeros((2, 1, 1), np.int32)) == E["BAD_SPECIES"]
    assert _code(n_species=17, epi=np.zeros((2, 17, 17), np.int32)) == E["BAD_SPECIES"]
    assert _code(n_shells=0) == E["BAD_SHELLS"]
    assert _code(n_shells=6, epi=make_epi(6, 4, 300, 1)) == E["BAD_SHELLS"]
    bad = make_epi(2, 4, 300, 1)
    bad[1, 0, 3] += 1
    assert _code(epi=bad) == E["EPI_NOT_SYMMETRIC"]
    assert _code(link_cell=1, dims=(16, 16, 16)) == E["LINK_CELL_TOO_SMALL"]   # 2w >= 2 r0 + R
    assert _code(n_shells=4, epi=make_epi(4, 4, 300, 1), link_cell=2, dims=(16, 16, 16)) == E["LINK_CELL_TOO_SMALL"]
    assert _code(accept=np.zeros(0, np.uint32)) == E["BAD_TABLE"]
    assert _code(storage=smcx.STORAGE_2BIT, kernel=smcx.KERNEL_WARP_PER_CELL) == E["UNSUPPORTED"]
    assert _code(lattice=1, n_shells=3, epi=make_epi(3, 4, 300, 1), kernel=smcx.KERNEL_THREAD_PER_CELL) == E["UNSUPPORTED"]
    # 4-bit storage belongs to the packed FCC / BCC kernels (the BCC one: two shells, link cell 4, <= 8 species)
    assert workspace_bytes(**_kw(storage=smcx.STORAGE_4BIT)) > 16 * 16 * 16                       # BCC, 2 shells: sweep_bcc4_thread
    assert _code(storage=smcx.STORAGE_4BIT, n_shells=1, epi=make_epi(1, 4, 300, 1)) == E["UNSUPPORTED"]
    assert _code(kernel=smcx.KERNEL_BCC4_THREAD, n_species=9, epi=make_epi(2, 9, 300, 1)) == E["UNSUPPORTED"]
    assert _code(kernel=smcx.KERNEL_BCC4_THREAD, storage=smcx.STORAGE_U8) == E["UNSUPPORTED"]
    fcc = dict(lattice=1, n_shells=3, n_species=5, epi=make_epi(3, 5, 400, 1))
    assert _code(storage=smcx.STORAGE_4BIT, kernel=smcx.KERNEL_GROUP_PER_CELL, **fcc) == E["UNSUPPORTED"]
    assert _code(kernel=smcx.KERNEL_FCC_THREAD, storage=smcx.STORAGE_U8, **fcc) == E["UNSUPPORTED"]
    assert _code(kernel=smcx.KERNEL_FCC_THREAD, lattice=1, n_shells=3, n_species=9, epi=make_epi(3, 9, 400, 1)) == E["UNSUPPORTED"]
    assert _code(kernel=smcx.KERNEL_FCC_THREAD, lattice=1, n_shells=3, n_species=5, epi=make_epi(3, 5, 20_000, 1)) == E["UNSUPPORTED"]
    assert _code(kernel=smcx.KERNEL_FCC_THREAD, dims=(16, 16, 16), link_cell=2, **fcc) == E["UNSUPPORTED"]
    n4 = workspace_bytes(**_kw(kernel=smcx.KERNEL_FCC_THREAD, dims=(32, 16, 16), **fcc))
    n8 = workspace_bytes(**_kw(kernel=smcx.KERNEL_GROUP_PER_CELL, dims=(32, 16, 16), **fcc))
    assert 0 < n8 - n4 <= 32 * 16 * 16 * 4 // 2 + 4096 and n4 >= 32 * 16 * 16 * 4 // 2
    assert workspace_bytes(**_kw(storage=smcx.STORAGE_4BIT, **fcc)) > 0                        # AUTO kernel follows the storage
    # explicit launch shape of the sub-warp kernel (smcx_params_t::group_lanes / group_warps; 0 = auto)
    assert _code(kernel=smcx.KERNEL_GROUP_PER_CELL, group_lanes=5) == E["UNSUPPORTED"]
    assert _code(kernel=smcx.KERNEL_GROUP_PER_CELL, group_lanes=64) == E["UNSUPPORTED"]
    assert _code(kernel=smcx.KERNEL_GROUP_PER_CELL, group_warps=9) == E["UNSUPPORTED"]
    assert _code(kernel=smcx.KERNEL_GROUP_PER_CELL, group_warps=-1) == E["UNSUPPORTED"]
    for lanes in (0, 4, 8, 16, 32):
        assert workspace_bytes(**_kw(kernel=smcx.KERNEL_GROUP_PER_CELL, group_lanes=lanes, group_warps=lanes // 8)) > 0
    # interactions so large that a trial's int32 dE could overflow
    huge = make_epi(2, 4, 300, 1) * 400_000
    assert _code(epi=huge) == E["EPI_RANGE"]
    assert _code(epi=huge, kernel=smcx.KERNEL_WARP_PER_CELL) == E["EPI_RANGE"]
    assert smcx.load_library().smcx_strerror(E["EPI_RANGE"]) != smcx.load_library().smcx_strerror(-99)
    # valid combinations pass
    assert workspace_bytes(**_kw()) > 0
    assert workspace_bytes(**_kw(n_shells=4, epi=make_epi(4, 4, 300, 1), link_cell=4, dims=(24, 16, 16))) > 0
    assert workspace_bytes(**_kw(lattice=1, n_shells=3, n_species=5, epi=make_epi(3, 5, 400, 1), link_cell=2,
                                 dims=(8, 8, 12))) > 0


def test_null_arguments_are_rejected_not_dereferenced():
    lib = smcx.load_library()
    assert lib.smcx_workspace_bytes(None, None) == E["NULL_ARG"]
    assert lib.smcx_create(None, None) == E["NULL_ARG"]
    assert lib.smcx_sweep(None, 1) == E["NULL_ARG"]
    assert lib.smcx_energy(None, None) == E["NULL_ARG"]
    lib.smcx_destroy(None)
    # replica ensemble
    assert lib.smcx_ensemble_create(None, None, 2, None, None, None, None, 0) == E["NULL_ARG"]
    assert lib.smcx_ensemble_sweep(None, 1) == E["NULL_ARG"]
    assert lib.smcx_ensemble_exchange(None, 0) == E["NULL_ARG"]
    assert lib.smcx_ensemble_run(None, 1, 1) == E["NULL_ARG"]
    assert lib.smcx_ensemble_state(None, None, None, None, None, None, None) == E["NULL_ARG"]
    assert lib.smcx_ensemble_replica(None, 0) is None
    assert lib.smcx_ensemble_kernel_launches(None) == 0
    lib.smcx_ensemble_destroy(None)


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(RuntimeError):
        smcx.Lattice(**_kw())
    # and straight through the C ABI: smcx_create must fail with SMCX_E_CUDA
    from paper_2509_20949_b200.binding import _make_params
    lib = smcx.load_library()
    p, keep = _make_params(kT_units=600, storage=0, kernel=0, device=0, trace_capacity=0, **_kw())
    h = C.c_void_p()
    assert lib.smcx_create(C.byref(h), C.byref(p)) == -11
    assert not h.value


@pytest.mark.parametrize("lat,dims,n_sp,n_shells,w", [
    (1, (128, 128, 128), 5, 3, 4),   # config 3
    (1, (400, 400, 400), 5, 3, 4),   # paper-shaped lattice (8 lanes)
    (0, (64, 64, 64), 5, 2, 4),      # BCC the thread kernels do not take
    (0, (24, 24, 24), 4, 4, 3),      # four shells, odd link cell
    (1, (16, 16, 16), 16, 5, 4),     # 78 neighbours, 16 species
])
def test_sub_warp_tile_layout_is_a_valid_one(lat, dims, n_sp, n_shells, w):
    """The layout group_tune_layout() picks on the host: every site of the (w + 2H)^3 tile gets an integral byte
    index of its own inside the tile, every neighbour sits in exactly one (lane, visit) slot, and the steps fit
    the 16 bits they are stored in."""
    from paper_2509_20949_b200.binding import group_layout
    from pygeom import shells
    forced = group_layout(lattice=lat, dims=dims, n_species=n_sp, n_shells=n_shells, epi=make_epi(n_shells, n_sp, 300, 1),
                          accept=make_accept_table(600), seed=1, link_cell=w, storage=smcx.STORAGE_U8, group_lanes=32)
    assert forced["lanes"] == 32                                            # the field is honoured
    L = group_layout(lattice=lat, dims=dims, n_species=n_sp, n_shells=n_shells, epi=make_epi(n_shells, n_sp, 300, 1),
                     accept=make_accept_table(600), seed=1, link_cell=w, storage=smcx.STORAGE_U8)
    assert L["lanes"] in (4, 8, 16, 32) and L["shift"] in (0, 1) and L["skew"] % 4 == 0
    sh, _ = shells(lat, n_shells)
    offs = np.concatenate(sh)                                              # (dx, dy, dz) per neighbour
    ZT = len(offs)
    slots = L["slots"]
    used = slots[slots != 255]
    assert sorted(used.tolist()) == list(range(ZT))
    visits = -(-ZT // L["lanes"])
    assert (slots[max(visits, 2 if visits <= 2 else 3 if visits <= 3 else 6 if visits <= 6 else visits) * L["lanes"]:] == 255).all()
    reach0 = np.abs(sh[0]).max()
    reach = np.abs(offs).max()
    H = (reach0 + reach + 1) // 2
    TW = w + 2 * H
    basis = [(0, 0, 0), (1, 1, 1)] if lat == 0 else [(0, 0, 0), (0, 1, 1), (1, 0, 1), (1, 1, 0)]
    t = np.arange(TW)
    tz, ty, tx = np.meshgrid(t, t, t, indexing="ij")
    idx = []
    for (bx, by, bz) in basis:
        num = (2 * tx + bx) + L["A"] * (2 * ty + by) + L["B"] * (2 * tz + bz)
        assert (num % (1 << L["shift"]) == 0).all()
        idx.append((num >> L["shift"]).ravel())
    idx = np.concatenate(idx)
    assert idx.min() >= 0 and idx.max() < L["tile_bytes"] and len(np.unique(idx)) == idx.size
    steps = (offs[:, 0] + L["A"] * offs[:, 1] + L["B"] * offs[:, 2])
    assert (steps % (1 << L["shift"]) == 0).all() and np.abs(steps >> L["shift"]).max() < 32768


def test_local_model_parameter_validation():
    """SMCX_MODEL_LOCAL (reading S12): its own link-cell bound (2w >= 2 r0 + 2R), at most 8 species, weights that keep the
    int32 dE of a trial exact, no slabs."""
    from smcx_inputs import make_local_weights
    w1, w2 = make_local_weights(2, 4, 200, 25, 1)
    ok = workspace_bytes(**_kw(epi=w1, local_quad=w2))
    assert ok > 16 * 16 * 16 * 2
    assert _code(epi=w1, local_quad=w2, link_cell=2) == E["LINK_CELL_TOO_SMALL"]      # fine for the pair model, not here
    assert workspace_bytes(**_kw(link_cell=2)) > 0
    w1b, w2b = make_local_weights(2, 9, 200, 25, 1)
    assert _code(n_species=9, epi=w1b, local_quad=w2b) == E["UNSUPPORTED"]
    assert _code(epi=w1, local_quad=w2 * 100000) == E["EPI_RANGE"]
    assert _code(epi=w1, local_quad=w2, kernel=smcx.KERNEL_GROUP_PER_CELL) == E["UNSUPPORTED"]
    assert _code(kernel=smcx.KERNEL_LOCAL_WARP) == E["UNSUPPORTED"]                     # that kernel serves the local model only
    info = smcx.domain_partition(2, 0, **_kw(dims=(16, 16, 32), epi=w1, local_quad=w2))
    assert info["ghost"] == 3 and info["z_layers"] == info["row_count"] * 4 + 3 + 6      # neighbours of neighbours


def test_header_is_c99_and_the_library_serves_a_plain_c_caller(tmp_path):
    """include/smcx.h compiles as C99 with -pedantic; a C program dlopens libsmcx.so and exercises the host-only calls."""
    import os
    import subprocess
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    hdr = os.path.join(root, "include", "smcx.h")
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Wextra", "-pedantic", "-Werror", "-fsyntax-only", "-x", "c", hdr])
    smcx.load_library()
    exe = str(tmp_path / "abi_from_c")
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Wextra", "-Werror", "-o", exe,
                           os.path.join(root, "tests", "host_checks", "abi_from_c.c"), "-ldl"])
    out = subprocess.run([exe, smcx.library_path()], capture_output=True, text=True)
    assert out.returncode == 0 and "abi_from_c ok" in out.stdout, out.stdout + out.stderr
