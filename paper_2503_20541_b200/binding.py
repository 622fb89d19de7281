"""Thin Python binding of libdimos_b200 (include/dimos.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels behind the C ABI; this module converts torch
tensors to raw pointers, hands the library torch's caching allocator and the current stream, and
turns status codes into exceptions.  There is no CPU fallback: if the shared library cannot be
loaded (or built with nvcc), importing the compute entry points fails loudly.

The three entry points keep the C names: `dimos_nl_build`, `dimos_nl_needs_rebuild`,
`dimos_nonbonded` (PAPER.md:173-185 NeighborHandling / get_neighborlist).
"""
from __future__ import annotations

import ctypes
import dataclasses
import os

import torch

from . import build_ext

DIMOS_F32, DIMOS_F64, DIMOS_MIXED = 0, 1, 2
DIMOS_RF, DIMOS_EWALD_REAL = 0, 1
UNIT = 8
_PRECISIONS = {"f32": DIMOS_F32, "f64": DIMOS_F64, "mixed": DIMOS_MIXED}
_METHODS = {"rf": DIMOS_RF, "ewald": DIMOS_EWALD_REAL}

EXPORTED_SYMBOLS = (
    "dimos_create", "dimos_destroy", "dimos_nl_build", "dimos_nl_destroy", "dimos_nl_needs_rebuild",
    "dimos_nonbonded", "dimos_nonbonded_host", "dimos_nl_export_pairs", "dimos_nl_stats", "dimos_launch_count",
    "dimos_probe_fp32_peak", "dimos_status_string", "dimos_last_error", "dimos_version",
    "dimos_nl_count_within", "dimos_profile_enable", "dimos_profile_read", "dimos_step_host", "dimos_nl_set_exceptions",
    "dimos_vv_kick_drift", "dimos_vv_kick", "dimos_nl_export_edges", "dimos_virtual_box",
    "dimos_dispersion_correction", "dimos_settle", "dimos_settle_velocities",
    "dimos_kinetic_energy", "dimos_berendsen", "dimos_water_kick_drift_settle", "dimos_water_kick_settle_velocities",
    "dimos_berendsen_scale", "dimos_pme_recip", "dimos_pme_mesh_size", "dimos_lj_table_fill", "dimos_langevin_ou",
    "dimos_nl_needs_rebuild_static",
)


class DimosError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"{message} (status {status})")
        self.status = status


class _Allocator(ctypes.Structure):
    _fields_ = [("alloc", ctypes.c_void_p), ("free_", ctypes.c_void_p), ("user", ctypes.c_void_p)]


class _Params(ctypes.Structure):
    _fields_ = [("r_cut", ctypes.c_double), ("eps_rf", ctypes.c_double), ("alpha", ctypes.c_double),
                ("coulomb_const", ctypes.c_double), ("method", ctypes.c_int32), ("r_switch", ctypes.c_double),
                ("skip_flag", ctypes.c_void_p)]


class _Stats(ctypes.Structure):
    _fields_ = [("n_atoms", ctypes.c_int64), ("n_units", ctypes.c_int64), ("n_slots", ctypes.c_int64),
                ("n_entries", ctypes.c_int64), ("n_entries_padded", ctypes.c_int64), ("n_pair_slots", ctypes.c_int64),
                ("list_bytes", ctypes.c_int64), ("workspace_bytes", ctypes.c_int64), ("n_cells", ctypes.c_int32 * 3),
                ("pbc_mode", ctypes.c_int32), ("row_capacity", ctypes.c_int32), ("n_rebuild_grow", ctypes.c_int32)]


_ALLOC_FN = ctypes.CFUNCTYPE(ctypes.c_void_p, ctypes.c_size_t, ctypes.c_void_p, ctypes.c_void_p)
_FREE_FN = ctypes.CFUNCTYPE(None, ctypes.c_void_p, ctypes.c_void_p)

_lib_handle = None


def library_path() -> str:
    return build_ext.OUT


def load_library() -> ctypes.CDLL:
    """Load libdimos_b200.so, building it in-tree with nvcc if it is missing or stale."""
    global _lib_handle
    if _lib_handle is not None:
        return _lib_handle
    path = build_ext.OUT
    if not os.path.exists(path) or build_ext._stale():
        try:
            build_ext.build()
        except Exception as exc:  # no silent fallback: the product IS the CUDA library
            if not os.path.exists(path):
                raise RuntimeError(f"libdimos_b200.so is missing and could not be built: {exc}") from exc
    lib = ctypes.CDLL(path)
    vp, i64, i32, dbl = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32, ctypes.c_double
    lib.dimos_create.argtypes = [ctypes.POINTER(vp), ctypes.c_int, ctypes.c_int, ctypes.POINTER(_Allocator)]
    lib.dimos_destroy.argtypes = [vp]
    lib.dimos_nl_build.argtypes = [vp, vp, i64, ctypes.POINTER(dbl), dbl, dbl, vp, i64, vp, vp, ctypes.POINTER(vp)]
    lib.dimos_nl_destroy.argtypes = [vp, vp]
    lib.dimos_nl_needs_rebuild.argtypes = [vp, vp, vp, i64, dbl, vp, ctypes.POINTER(i32), vp]
    lib.dimos_nl_needs_rebuild_static.argtypes = [vp, vp, vp, i64, dbl, vp, vp, vp]
    lib.dimos_nonbonded.argtypes = [vp, vp, vp, vp, vp, vp, i32, ctypes.POINTER(dbl), ctypes.POINTER(_Params), vp, vp, vp, vp]
    lib.dimos_nonbonded_host.argtypes = [vp, vp, vp, vp, vp, vp, i32, ctypes.POINTER(dbl), ctypes.POINTER(_Params), vp, vp, vp, vp]
    lib.dimos_nl_export_pairs.argtypes = [vp, vp, vp, i64, ctypes.POINTER(i64), vp]
    lib.dimos_step_host.argtypes = [vp, ctypes.POINTER(vp), vp, vp, vp, vp, i32, i64, ctypes.POINTER(dbl), dbl, vp, i64,
                                    ctypes.POINTER(_Params), vp, vp, vp, ctypes.POINTER(i32), vp]
    lib.dimos_step_host.restype = ctypes.c_int
    lib.dimos_nl_count_within.argtypes = [vp, vp, dbl, ctypes.POINTER(i64), vp]
    lib.dimos_nl_set_exceptions.argtypes = [vp, vp, vp, vp, i64, vp]
    lib.dimos_vv_kick_drift.argtypes = [vp, vp, vp, vp, vp, i64, dbl, vp, dbl, vp, ctypes.POINTER(i32), vp]
    lib.dimos_vv_kick.argtypes = [vp, vp, vp, vp, i64, dbl, vp, vp]
    lib.dimos_settle.argtypes = [vp, vp, vp, vp, vp, i64, dbl, dbl, dbl, dbl, dbl, vp]
    lib.dimos_settle_velocities.argtypes = [vp, vp, vp, vp, i64, dbl, dbl, vp]
    lib.dimos_water_kick_drift_settle.argtypes = [vp, vp, vp, vp, vp, i64, dbl, dbl, dbl, dbl, dbl, vp, dbl, vp,
                                                  ctypes.POINTER(i32), vp]
    lib.dimos_water_kick_settle_velocities.argtypes = [vp, vp, vp, vp, vp, i64, dbl, dbl, dbl, vp, vp, vp]
    lib.dimos_berendsen_scale.argtypes = [vp, vp, i64, i64, dbl, dbl, dbl, vp, vp]
    lib.dimos_kinetic_energy.argtypes = [vp, vp, vp, i64, vp, ctypes.POINTER(dbl), vp]
    lib.dimos_berendsen.argtypes = [vp, vp, vp, i64, i64, dbl, dbl, dbl, vp, ctypes.POINTER(dbl), vp]
    lib.dimos_nl_export_edges.argtypes = [vp, vp, dbl, vp, vp, vp, i64, ctypes.POINTER(i64), vp]
    lib.dimos_virtual_box.argtypes = [vp, vp, i64, dbl, dbl, ctypes.POINTER(dbl), ctypes.POINTER(dbl), vp]
    lib.dimos_dispersion_correction.argtypes = [vp, vp, i64, vp, i32, ctypes.POINTER(dbl), dbl, dbl, ctypes.POINTER(dbl),
                                                ctypes.POINTER(dbl), vp]
    lib.dimos_pme_recip.argtypes = [vp, vp, vp, i64, ctypes.POINTER(dbl), dbl, ctypes.POINTER(i32), i32, dbl, vp, i32, vp, vp, vp]
    lib.dimos_pme_mesh_size.argtypes = [dbl, ctypes.POINTER(dbl), dbl, ctypes.POINTER(i32)]
    lib.dimos_lj_table_fill.argtypes = [vp, vp, i32, vp]
    lib.dimos_langevin_ou.argtypes = [vp, vp, vp, vp, i64, dbl, dbl, dbl, vp]
    lib.dimos_profile_enable.argtypes = [vp, ctypes.c_int]
    lib.dimos_profile_read.argtypes = [vp, ctypes.POINTER(dbl), ctypes.POINTER(i64)]
    lib.dimos_nl_stats.argtypes = [vp, ctypes.POINTER(_Stats)]
    lib.dimos_launch_count.argtypes = [vp]
    lib.dimos_launch_count.restype = i64
    lib.dimos_probe_fp32_peak.argtypes = [vp, dbl, ctypes.POINTER(dbl), vp]
    lib.dimos_status_string.argtypes = [ctypes.c_int]
    lib.dimos_status_string.restype = ctypes.c_char_p
    lib.dimos_last_error.argtypes = [vp]
    lib.dimos_last_error.restype = ctypes.c_char_p
    lib.dimos_version.restype = ctypes.c_char_p
    for name in ("dimos_create", "dimos_destroy", "dimos_nl_build", "dimos_nl_destroy", "dimos_nl_needs_rebuild",
                 "dimos_nonbonded", "dimos_nonbonded_host", "dimos_nl_export_pairs", "dimos_nl_stats",
                 "dimos_probe_fp32_peak", "dimos_nl_count_within", "dimos_profile_enable", "dimos_profile_read",
                 "dimos_nl_set_exceptions", "dimos_vv_kick_drift", "dimos_vv_kick", "dimos_nl_export_edges", "dimos_virtual_box", "dimos_dispersion_correction",
                 "dimos_settle", "dimos_settle_velocities", "dimos_kinetic_energy", "dimos_berendsen",
                 "dimos_water_kick_drift_settle", "dimos_water_kick_settle_velocities", "dimos_berendsen_scale",
                 "dimos_pme_recip", "dimos_pme_mesh_size", "dimos_lj_table_fill", "dimos_langevin_ou"):
        getattr(lib, name).restype = ctypes.c_int
    _lib_handle = lib
    return lib


def _stream_ptr() -> int:
    return int(torch.cuda.current_stream().cuda_stream)


def _box3(box):
    vals = [float(b) for b in (box.tolist() if hasattr(box, "tolist") else box)]
    if len(vals) != 3:
        raise ValueError("box must have 3 entries")
    return (ctypes.c_double * 3)(*vals)


@dataclasses.dataclass
class NeighborList:
    handle: ctypes.c_void_p
    ctx: "Context"
    pos_at_build: torch.Tensor
    box: tuple
    r_cut: float
    skin: float

    def stats(self) -> dict:
        return self.ctx.nl_stats(self)


class Context:
    """One library context: device + precision + torch-backed allocator."""

    def __init__(self, device: int = 0, precision: str = "f32", torch_allocator: bool = True, guard_bytes: int = 0):
        """guard_bytes > 0 (a multiple of 256): every workspace block the library asks for is allocated with that many
        bytes of 0xA5 in front of and behind it; check_guards() reports blocks whose guards were overwritten (the
        out-of-bounds-write check of tests/test_gpu_guards.py; compute-sanitizer is not available on every pool)."""
        if not torch.cuda.is_available():
            raise RuntimeError("dimos_b200 needs a CUDA device: there is no CPU fallback")
        self.lib = load_library()
        self.device = int(device)
        self.precision = precision
        self.real = torch.float64 if precision == "f64" else torch.float32
        self._blocks: dict[int, torch.Tensor] = {}
        self._alloc_struct = None
        self._guard = int(guard_bytes)
        self._guard_violations: list[tuple[int, int]] = []
        self.fail_alloc_after: int | None = None  # tests: the allocator callback succeeds this many more times, then returns NULL
        if self._guard % 256 != 0:
            raise ValueError("guard_bytes must be a multiple of 256")
        if torch_allocator:
            dev = torch.device("cuda", self.device)

            def _alloc(nbytes, _stream, _user):
                g = self._guard
                if self.fail_alloc_after is not None:  # fault injection for the error-path tests
                    if self.fail_alloc_after <= 0:
                        return None
                    self.fail_alloc_after -= 1
                try:
                    t = torch.empty(int(nbytes) + 2 * g, dtype=torch.uint8, device=dev)
                    if g:
                        t[:g] = 0xA5
                        t[g + int(nbytes):] = 0xA5
                except Exception:
                    return None
                self._blocks[t.data_ptr() + g] = t
                return t.data_ptr() + g

            def _free(ptr, _user):
                t = self._blocks.pop(int(ptr), None)
                if t is not None and self._guard:
                    self._check_block(int(ptr), t)

            self._alloc_cb = _ALLOC_FN(_alloc)
            self._free_cb = _FREE_FN(_free)
            self._alloc_struct = _Allocator(ctypes.cast(self._alloc_cb, ctypes.c_void_p),
                                            ctypes.cast(self._free_cb, ctypes.c_void_p), None)
        h = ctypes.c_void_p()
        with torch.cuda.device(self.device):
            rc = self.lib.dimos_create(ctypes.byref(h), self.device, _PRECISIONS[precision],
                                       ctypes.byref(self._alloc_struct) if self._alloc_struct else None)
        if rc != 0:
            raise DimosError(rc, self.lib.dimos_status_string(rc).decode())
        self.handle = h
        self._flag = torch.zeros(1, dtype=torch.int32, device=torch.device("cuda", self.device))

    # -- helpers ---------------------------------------------------------------------------------
    def _check(self, rc: int):
        if rc != 0:
            msg = self.lib.dimos_last_error(self.handle).decode() or self.lib.dimos_status_string(rc).decode()
            raise DimosError(rc, msg)

    def _dev(self, t: torch.Tensor, dtype, shape_last=None) -> torch.Tensor:
        if not t.is_cuda or t.dtype != dtype or not t.is_contiguous():
            raise ValueError(f"expected a contiguous CUDA tensor of dtype {dtype}, got {t.dtype} on {t.device}")
        if shape_last is not None and (t.dim() != 2 or t.shape[1] != shape_last):
            raise ValueError(f"expected shape (N, {shape_last})")
        return t

    def _check_block(self, ptr: int, t: torch.Tensor):
        g = self._guard
        torch.cuda.synchronize(self.device)
        bad = int((t[:g] != 0xA5).sum()) + int((t[t.numel() - g:] != 0xA5).sum())
        if bad:
            self._guard_violations.append((t.numel() - 2 * g, bad))

    def check_guards(self) -> list:
        """(block size, overwritten guard bytes) of every workspace block, live or freed, whose guards were touched."""
        if not self._guard:
            raise RuntimeError("context was created without guard_bytes")
        live = list(self._guard_violations)
        for ptr, t in self._blocks.items():
            before = len(self._guard_violations)
            self._check_block(ptr, t)
            live += self._guard_violations[before:]
            del self._guard_violations[before:]
        return live

    def close(self):
        if getattr(self, "handle", None):
            torch.cuda.synchronize(self.device)
            self.lib.dimos_destroy(self.handle)
            self.handle = None
            self._blocks.clear()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()
        return False

    # -- the C-ABI calls -------------------------------------------------------------------------
    def nl_build(self, pos, box, r_cut, skin, excl_pairs=None, pos_at_build=None, nl: NeighborList | None = None):
        """dimos_nl_build: returns a NeighborList (rebuilt in place when `nl` is given)."""
        pos = self._dev(pos, self.real, 3)
        n = pos.shape[0]
        if pos_at_build is None:
            pos_at_build = nl.pos_at_build if nl is not None and nl.pos_at_build.shape == pos.shape else torch.empty_like(pos)
        self._dev(pos_at_build, self.real, 3)
        n_excl = 0
        excl_ptr = None
        if excl_pairs is not None and excl_pairs.numel() > 0:
            excl_pairs = self._dev(excl_pairs, torch.int32, 2)
            n_excl = excl_pairs.shape[0]
            excl_ptr = excl_pairs.data_ptr()
        h = ctypes.c_void_p(nl.handle.value if nl is not None else None)
        with torch.cuda.device(self.device):
            rc = self.lib.dimos_nl_build(self.handle, pos.data_ptr(), n, _box3(box), float(r_cut), float(skin), excl_ptr,
                                         n_excl, pos_at_build.data_ptr(), _stream_ptr(), ctypes.byref(h))
        self._check(rc)
        boxt = tuple(float(b) for b in (box.tolist() if hasattr(box, "tolist") else box))
        if nl is not None:
            nl.handle, nl.pos_at_build, nl.box, nl.r_cut, nl.skin = h, pos_at_build, boxt, float(r_cut), float(skin)
            return nl
        return NeighborList(h, self, pos_at_build, boxt, float(r_cut), float(skin))

    def nl_needs_rebuild(self, pos, pos_at_build, skin, sync: bool = True, flag=None):
        """dimos_nl_needs_rebuild: bool when sync=True, else the device flag tensor (no host sync)."""
        pos = self._dev(pos, self.real, 3)
        ref = self._dev(pos_at_build, self.real, 3)
        host = ctypes.c_int32(0)
        with torch.cuda.device(self.device):
            rc = self.lib.dimos_nl_needs_rebuild(self.handle, pos.data_ptr(), ref.data_ptr(), pos.shape[0], float(skin),
                                                 (flag if flag is not None else self._flag).data_ptr(),
                                                 ctypes.byref(host) if sync else None, _stream_ptr())
        self._check(rc)
        return bool(host.value) if sync else (flag if flag is not None else self._flag)

    def nl_needs_rebuild_static(self, pos, pos_at_build, skin, flag, max_disp2=None):
        """dimos_nl_needs_rebuild_static: the trigger with its scratch in a fixed device array (no allocation, no host
        synchronisation).  flag: int32 device tensor (required, caller-owned); max_disp2: float64 device tensor or None."""
        pos = self._dev(pos, self.real, 3)
        ref = self._dev(pos_at_build, self.real, 3)
        flag = self._dev(flag, torch.int32)
        if max_disp2 is not None:
            max_disp2 = self._dev(max_disp2, torch.float64)
        with torch.cuda.device(self.device):
            rc = self.lib.dimos_nl_needs_rebuild_static(self.handle, pos.data_ptr(), ref.data_ptr(), pos.shape[0], float(skin),
                                                        flag.data_ptr(), max_disp2.data_ptr() if max_disp2 is not None else None,
                                                        _stream_ptr())
        self._check(rc)
        return flag

    def _params(self, nl, method, eps_rf, alpha, coulomb_const, r_switch=0.0, skip_flag=None):
        skip = None
        if skip_flag is not None:
            if not skip_flag.is_cuda or skip_flag.dtype != torch.int32 or skip_flag.numel() < 1:
                raise ValueError("skip_flag must be an int32 device tensor")
            skip = skip_flag.data_ptr()
        return _Params(float(nl.r_cut), float(eps_rf), float(alpha), float(coulomb_const),
                       _METHODS[method] if isinstance(method, str) else int(method), float(r_switch), skip)

    def nonbonded(self, nl: NeighborList, pos, charge, type_, lj_table, *, method="rf", eps_rf=78.5, alpha=3.12,
                  coulomb_const=138.935456, r_switch=0.0, F=None, E=None, virial=None, skip_flag=None):
        """dimos_nonbonded: returns (F (N,3) real, E (4,) float64, virial (3,3) float64) device tensors.
        skip_flag: dimos_nb_params.skip_flag, an int32 device tensor (the kernels do nothing if it is non-zero when they run)."""
        pos = self._dev(pos, self.real, 3)
        n = pos.shape[0]
        charge = self._dev(charge, self.real)
        type_ = self._dev(type_, torch.int32)
        lj_table = self._dev(lj_table, torch.float64)
        nt = lj_table.shape[0]
        if lj_table.shape != (nt, nt, 2) or charge.numel() != n or type_.numel() != n:
            raise ValueError("shape mismatch")
        dev = pos.device
        F = torch.empty_like(pos) if F is None else self._dev(F, self.real, 3)
        E = torch.empty(4, dtype=torch.float64, device=dev) if E is None else self._dev(E, torch.float64)
        virial = torch.empty(3, 3, dtype=torch.float64, device=dev) if virial is None else self._dev(virial, torch.float64)
        prm = self._params(nl, method, eps_rf, alpha, coulomb_const, r_switch, skip_flag)
        with torch.cuda.device(self.device):
            rc = self.lib.dimos_nonbonded(self.handle, nl.handle, pos.data_ptr(), charge.data_ptr(), type_.data_ptr(),
                                          lj_table.data_ptr(), nt, _box3(nl.box), ctypes.byref(prm), F.data_ptr(),
                                          E.data_ptr(), virial.data_ptr(), _stream_ptr())
        self._check(rc)
        return F, E, virial

    def nonbonded_host(self, nl: NeighborList, pos, charge, type_, lj_table, F, E, virial, *, method="rf", eps_rf=78.5,
                       alpha=3.12, coulomb_const=138.935456, r_switch=0.0):
        """dimos_nonbonded_host: all arrays are HOST tensors (pinned recommended); synchronises."""
        for t in (pos, charge, type_, lj_table, F, E, virial):
            if t.is_cuda or not t.is_contiguous():
                raise ValueError("nonbonded_host takes contiguous host tensors")
        prm = self._params(nl, method, eps_rf, alpha, coulomb_const, r_switch)
        with torch.cuda.device(self.device):
            rc = self.lib.dimos_nonbonded_host(self.handle, nl.handle, pos.data_ptr(), charge.data_ptr(), type_.data_ptr(),
                                               lj_table.data_ptr(), lj_table.shape[0], _box3(nl.box), ctypes.byref(prm),
                                               F.data_ptr(), E.data_ptr(), virial.data_ptr(), _stream_ptr())
        self._check(rc)
        return F, E, virial

    def step_host(self, nl: "NeighborList | None", pos, charge, type_, lj_table, box, r_cut, skin, excl_pairs, F, E, virial, *,
                  method="rf", eps_rf=78.5, alpha=3.12, coulomb_const=138.935456, r_switch=0.0, ntypes=None):
        """dimos_step_host: HOST tensors in and out; returns (NeighborList, rebuilt: bool).  charge / type_ / lj_table may be
        None after a call on this list has passed them (the list keeps its device copies); give ntypes then."""
        for t in (pos, charge, type_, lj_table, F, E, virial, excl_pairs):
            if t is not None and (t.is_cuda or not t.is_contiguous()):
                raise ValueError("step_host takes contiguous host tensors")
        prm = _Params(float(r_cut), float(eps_rf), float(alpha), float(coulomb_const), _METHODS[method], float(r_switch), None)
        h = ctypes.c_void_p(nl.handle.value if nl is not None else None)
        rebuilt = ctypes.c_int32(0)
        n_excl = 0 if excl_pairs is None else excl_pairs.shape[0]
        nt = lj_table.shape[0] if lj_table is not None else int(ntypes)
        ptr = lambda t: t.data_ptr() if t is not None else None
        with torch.cuda.device(self.device):
            rc = self.lib.dimos_step_host(self.handle, ctypes.byref(h), pos.data_ptr(), ptr(charge), ptr(type_), ptr(lj_table), nt,
                                          pos.shape[0], _box3(box), float(skin), excl_pairs.data_ptr() if n_excl else None, n_excl,
                                          ctypes.byref(prm), F.data_ptr(), E.data_ptr(), virial.data_ptr(), ctypes.byref(rebuilt),
                                          _stream_ptr())
        self._check(rc)
        boxt = tuple(float(b) for b in (box.tolist() if hasattr(box, "tolist") else box))
        if nl is None:
            nl = NeighborList(h, self, torch.empty(0), boxt, float(r_cut), float(skin))
        else:
            nl.handle = h
        return nl, bool(rebuilt.value)

    def pme_recip(self, pos, charge, box, alpha, mesh, order=5, coulomb_const=138.935456, F=None, accumulate=False,
                  want_forces=True, E=None, virial=None):
        """dimos_pme_recip: (F (N,3) or None, E (2,) = {U_recip, U_self}, virial (3,3)) device tensors; no sync."""
        real = torch.float64 if self.precision == "f64" else torch.float32
        pos = self._dev(pos, real, 3)
        charge = self._dev(charge, real)
        n = pos.shape[0]
        if F is None and want_forces:
            F = torch.zeros((n, 3), dtype=real, device=pos.device) if accumulate else torch.empty((n, 3), dtype=real, device=pos.device)
        if E is None:
            E = torch.empty(2, dtype=torch.float64, device=pos.device)
        if virial is None:
            virial = torch.empty((3, 3), dtype=torch.float64, device=pos.device)
        m = (ctypes.c_int32 * 3)(*[int(k) for k in mesh])
        with torch.cuda.device(self.device):
            rc = self.lib.dimos_pme_recip(self.handle, pos.data_ptr(), charge.data_ptr(), n, _box3(box), float(alpha), m, int(order),
                                          float(coulomb_const), F.data_ptr() if F is not None else None, 1 if accumulate else 0,
                                          E.data_ptr(), virial.data_ptr(), _stream_ptr())
        self._check(rc)
        return F, E, virial

    def dispersion_correction(self, type_, lj_table, box, r_cut, r_switch=0.0):
        """dimos_dispersion_correction: (E float, virial (3,3) float64 numpy) of the LJ tail correction."""
        import numpy as np

        type_ = self._dev(type_, torch.int32)
        lj_table = self._dev(lj_table, torch.float64)
        e = ctypes.c_double(0.0)
        w = (ctypes.c_double * 9)()
        with torch.cuda.device(self.device):
            rc = self.lib.dimos_dispersion_correction(self.handle, type_.data_ptr(), type_.numel(), lj_table.data_ptr(),
                                                      lj_table.shape[0], _box3(box), float(r_cut), float(r_switch),
                                                      ctypes.byref(e), w, _stream_ptr())
        self._check(rc)
        return float(e.value), np.array(list(w), dtype=np.float64).reshape(3, 3)

    def virtual_box(self, pos, r_cut, skin):
        """dimos_virtual_box: (box (3,) float64 numpy, lower corner (3,)) of the virtual periodic box of an open system."""
        import numpy as np

        pos = self._dev(pos, self.real, 3)
        box = (ctypes.c_double * 3)()
        lo = (ctypes.c_double * 3)()
        with torch.cuda.device(self.device):
            rc = self.lib.dimos_virtual_box(self.handle, pos.data_ptr(), pos.shape[0], float(r_cut), float(skin), box, lo,
                                            _stream_ptr())
        self._check(rc)
        return np.array(list(box), dtype=np.float64), np.array(list(lo), dtype=np.float64)

    def vv_kick_drift(self, pos, vel, F, inv_mass, dt, pos_at_build=None, skin=0.0, sync=True, flag=None):
        """dimos_vv_kick_drift: velocity-Verlet steps 1 + 2 in place; with pos_at_build also the rebuild flag (bool when
        sync, else the device flag tensor)."""
        pos = self._dev(pos, self.real, 3)
        vel = self._dev(vel, self.real, 3)
        F = self._dev(F, self.real, 3)
        inv_mass = self._dev(inv_mass, self.real)
        host = ctypes.c_int32(0)
        trig = pos_at_build is not None
        flag = self._flag if flag is None else self._dev(flag, torch.int32)  # the device word that receives the trigger's result
        if trig:
            pos_at_build = self._dev(pos_at_build, self.real, 3)
        with torch.cuda.device(self.device):
            rc = self.lib.dimos_vv_kick_drift(self.handle, pos.data_ptr(), vel.data_ptr(), F.data_ptr(), inv_mass.data_ptr(),
                                              pos.shape[0], float(dt), pos_at_build.data_ptr() if trig else None, float(skin),
                                              flag.data_ptr() if trig else None,
                                              ctypes.byref(host) if (trig and sync) else None, _stream_ptr())
        self._check(rc)
        if not trig:
            return None
        return bool(host.value) if sync else flag

    def _skip_ptr(self, skip_flag):
        if skip_flag is None:
            return None
        if not skip_flag.is_cuda or skip_flag.dtype != torch.int32 or skip_flag.numel() < 1:
            raise ValueError("skip_flag must be an int32 device tensor")
        return skip_flag.data_ptr()

    def vv_kick(self, vel, F, inv_mass, dt, skip_flag=None):
        """dimos_vv_kick: velocity-Verlet step 5 in place (not at all if the device word skip_flag is non-zero)."""
        vel = self._dev(vel, self.real, 3)
        F = self._dev(F, self.real, 3)
        inv_mass = self._dev(inv_mass, self.real)
        with torch.cuda.device(self.device):
            rc = self.lib.dimos_vv_kick(self.handle, vel.data_ptr(), F.data_ptr(), inv_mass.data_ptr(), vel.shape[0], float(dt),
                                        self._skip_ptr(skip_flag), _stream_ptr())
        self._check(rc)

    def langevin_ou(self, vel, inv_mass, xi, gamma, dt, T):
        """dimos_langevin_ou: exact Ornstein-Uhlenbeck velocity update in place on vel with the caller's normal numbers xi."""
        vel = self._dev(vel, self.real, 3)
        inv_mass = self._dev(inv_mass, self.real)
        xi = self._dev(xi, self.real, 3)
        with torch.cuda.device(self.device):
            rc = self.lib.dimos_langevin_ou(self.handle, vel.data_ptr(), inv_mass.data_ptr(), xi.data_ptr(), vel.shape[0], float(gamma),
                                            float(dt), float(T), _stream_ptr())
        self._check(rc)

    def settle(self, pos_old, pos, water, m_O, m_H, d_OH, d_HH, vel=None, dt=0.0):
        """dimos_settle: rigid-water position constraints (velocity-Verlet step 3) in place on pos (and vel if given)."""
        pos_old = self._dev(pos_old, self.real, 3)
        pos = self._dev(pos, self.real, 3)
        water = self._dev(water, torch.int32, 3)
        if vel is not None:
            vel = self._dev(vel, self.real, 3)
        with torch.cuda.device(self.device):
            rc = self.lib.dimos_settle(self.handle, pos_old.data_ptr(), pos.data_ptr(), vel.data_ptr() if vel is not None else None,
                                       water.data_ptr(), water.shape[0], float(m_O), float(m_H), float(d_OH), float(d_HH),
                                       float(dt), _stream_ptr())
        self._check(rc)

    def settle_velocities(self, pos, vel, water, m_O, m_H):
        """dimos_settle_velocities: rigid-water velocity constraints (velocity-Verlet step 6) in place on vel."""
        pos = self._dev(pos, self.real, 3)
        vel = self._dev(vel, self.real, 3)
        water = self._dev(water, torch.int32, 3)
        with torch.cuda.device(self.device):
            rc = self.lib.dimos_settle_velocities(self.handle, pos.data_ptr(), vel.data_ptr(), water.data_ptr(), water.shape[0],
                                                  float(m_O), float(m_H), _stream_ptr())
        self._check(rc)

    def water_kick_drift_settle(self, pos, vel, F, water, m_O, m_H, d_OH, d_HH, dt, pos_at_build=None, skin=0.0, sync=True,
                                flag=None):
        """dimos_water_kick_drift_settle: steps 1 + 2 + 3 for rigid waters in one pass; returns the rebuild flag like
        vv_kick_drift (None without pos_at_build)."""
        pos = self._dev(pos, self.real, 3)
        vel = self._dev(vel, self.real, 3)
        F = self._dev(F, self.real, 3)
        water = self._dev(water, torch.int32, 3)
        host = ctypes.c_int32(0)
        trig = pos_at_build is not None
        flag = self._flag if flag is None else self._dev(flag, torch.int32)  # the device word that receives the trigger's result
        if trig:
            pos_at_build = self._dev(pos_at_build, self.real, 3)
        with torch.cuda.device(self.device):
            rc = self.lib.dimos_water_kick_drift_settle(
                self.handle, pos.data_ptr(), vel.data_ptr(), F.data_ptr(), water.data_ptr(), water.shape[0], float(m_O),
                float(m_H), float(d_OH), float(d_HH), float(dt), pos_at_build.data_ptr() if trig else None, float(skin),
                flag.data_ptr() if trig else None, ctypes.byref(host) if (trig and sync) else None, _stream_ptr())
        self._check(rc)
        if not trig:
            return None
        return bool(host.value) if sync else flag

    def water_kick_settle_velocities(self, pos, vel, F, water, m_O, m_H, dt, want_ke=False, skip_flag=None):
        """dimos_water_kick_settle_velocities: steps 5 + 6 for rigid waters in one pass; with want_ke returns the device
        tensor (1 double) that receives the kinetic energy of the constrained velocities."""
        pos = self._dev(pos, self.real, 3)
        vel = self._dev(vel, self.real, 3)
        F = self._dev(F, self.real, 3)
        water = self._dev(water, torch.int32, 3)
        ke = self._ke_scratch() if want_ke else None
        with torch.cuda.device(self.device):
            rc = self.lib.dimos_water_kick_settle_velocities(self.handle, pos.data_ptr(), vel.data_ptr(), F.data_ptr(),
                                                             water.data_ptr(), water.shape[0], float(m_O), float(m_H), float(dt),
                                                             ke.data_ptr() if want_ke else None, self._skip_ptr(skip_flag),
                                                             _stream_ptr())
        self._check(rc)
        return ke

    def _ke_scratch(self):
        if getattr(self, "_ke", None) is None:
            self._ke = torch.zeros(1, dtype=torch.float64, device=self.device)
        return self._ke

    def kinetic_energy(self, vel, inv_mass) -> float:
        """dimos_kinetic_energy: K = 1/2 sum m v^2 in kJ/mol (synchronises)."""
        vel = self._dev(vel, self.real, 3)
        inv_mass = self._dev(inv_mass, self.real)
        out = ctypes.c_double(0.0)
        with torch.cuda.device(self.device):
            rc = self.lib.dimos_kinetic_energy(self.handle, vel.data_ptr(), inv_mass.data_ptr(), vel.shape[0],
                                               self._ke_scratch().data_ptr(), ctypes.byref(out), _stream_ptr())
        self._check(rc)
        return out.value

    def berendsen(self, vel, inv_mass, n_dof, T0, tau, dt, sync=True):
        """dimos_berendsen: rescale vel in place; returns the temperature before the scaling (None with sync=False)."""
        vel = self._dev(vel, self.real, 3)
        inv_mass = self._dev(inv_mass, self.real)
        out = ctypes.c_double(0.0)
        with torch.cuda.device(self.device):
            rc = self.lib.dimos_berendsen(self.handle, vel.data_ptr(), inv_mass.data_ptr(), vel.shape[0], int(n_dof), float(T0),
                                          float(tau), float(dt), self._ke_scratch().data_ptr(),
                                          ctypes.byref(out) if sync else None, _stream_ptr())
        self._check(rc)
        return out.value if sync else None

    def berendsen_scale(self, vel, n_dof, T0, tau, dt, ke):
        """dimos_berendsen_scale: rescale vel with the kinetic energy already in the device tensor `ke` (1 double)."""
        vel = self._dev(vel, self.real, 3)
        ke = self._dev(ke, torch.float64)
        with torch.cuda.device(self.device):
            rc = self.lib.dimos_berendsen_scale(self.handle, vel.data_ptr(), vel.shape[0], int(n_dof), float(T0), float(tau),
                                                float(dt), ke.data_ptr(), _stream_ptr())
        self._check(rc)

    def nl_set_exceptions(self, nl: NeighborList, pairs, scale):
        """dimos_nl_set_exceptions: pairs (n,2) int32 i<j, scale (n,2) float64 = (Coulomb scale, LJ scale); None clears."""
        if pairs is None or len(pairs) == 0:
            with torch.cuda.device(self.device):
                rc = self.lib.dimos_nl_set_exceptions(self.handle, nl.handle, None, None, 0, _stream_ptr())
            self._check(rc)
            return
        pairs = self._dev(pairs, torch.int32, 2)
        scale = self._dev(scale, torch.float64, 2)
        if pairs.shape[0] != scale.shape[0]:
            raise ValueError("exceptions: pairs and scales differ in length")
        with torch.cuda.device(self.device):
            rc = self.lib.dimos_nl_set_exceptions(self.handle, nl.handle, pairs.data_ptr(), scale.data_ptr(), pairs.shape[0],
                                                  _stream_ptr())
        self._check(rc)

    def nl_export_pairs(self, nl: NeighborList) -> torch.Tensor:
        """dimos_nl_export_pairs: (n,2) int32 device tensor of pairs i<j, order unspecified."""
        n = ctypes.c_int64(0)
        with torch.cuda.device(self.device):
            rc = self.lib.dimos_nl_export_pairs(self.handle, nl.handle, None, 0, ctypes.byref(n), _stream_ptr())
        self._check(rc)
        out = torch.empty((max(n.value, 1), 2), dtype=torch.int32, device=torch.device("cuda", self.device))
        got = ctypes.c_int64(0)
        with torch.cuda.device(self.device):
            rc = self.lib.dimos_nl_export_pairs(self.handle, nl.handle, out.data_ptr(), out.shape[0], ctypes.byref(got), _stream_ptr())
        self._check(rc)
        return out[: got.value]

    def nl_export_edges(self, nl: NeighborList, radius: float):
        """dimos_nl_export_edges: (pairs (n,2) int32 a<b, dvec (n,3) real = r_a - r_b - shift*box, shift (n,3) int32) of the
        pairs with minimum-image r < radius at the build positions; device tensors, order unspecified."""
        n = self.nl_count_within(nl, radius)
        dev = torch.device("cuda", self.device)
        pairs = torch.empty((max(n, 1), 2), dtype=torch.int32, device=dev)
        dvec = torch.empty((max(n, 1), 3), dtype=self.real, device=dev)
        shift = torch.empty((max(n, 1), 3), dtype=torch.int32, device=dev)
        got = ctypes.c_int64(0)
        with torch.cuda.device(self.device):
            rc = self.lib.dimos_nl_export_edges(self.handle, nl.handle, float(radius), pairs.data_ptr(), dvec.data_ptr(),
                                                shift.data_ptr(), pairs.shape[0], ctypes.byref(got), _stream_ptr())
        self._check(rc)
        return pairs[: got.value], dvec[: got.value], shift[: got.value]

    def nl_count_within(self, nl: NeighborList, radius: float) -> int:
        """dimos_nl_count_within: pairs of the list with r < radius at the build positions."""
        n = ctypes.c_int64(0)
        with torch.cuda.device(self.device):
            rc = self.lib.dimos_nl_count_within(self.handle, nl.handle, float(radius), ctypes.byref(n), _stream_ptr())
        self._check(rc)
        return int(n.value)

    def profile_enable(self, on: bool = True):
        self._check(self.lib.dimos_profile_enable(self.handle, 1 if on else 0))

    def profile_read(self):
        """(summed pair-force kernel milliseconds, launches covered) since the last read."""
        ms, n = ctypes.c_double(0.0), ctypes.c_int64(0)
        self._check(self.lib.dimos_profile_read(self.handle, ctypes.byref(ms), ctypes.byref(n)))
        return float(ms.value), int(n.value)

    def nl_stats(self, nl: NeighborList) -> dict:
        st = _Stats()
        rc = self.lib.dimos_nl_stats(nl.handle, ctypes.byref(st))
        self._check(rc)
        d = {name: getattr(st, name) for name, _ in _Stats._fields_ if name != "n_cells"}
        d["n_cells"] = tuple(st.n_cells)
        return d

    def launch_count(self) -> int:
        return int(self.lib.dimos_launch_count(self.handle))

    def probe_fp32_peak(self, ms_target: float = 3.0) -> float:
        out = ctypes.c_double(0.0)
        with torch.cuda.device(self.device):
            rc = self.lib.dimos_probe_fp32_peak(self.handle, float(ms_target), ctypes.byref(out), _stream_ptr())
        self._check(rc)
        return float(out.value)


# -- module-level functions with the C names -------------------------------------------------------
def dimos_nl_build(ctx: Context, pos, box, r_cut, skin, excl_pairs=None, pos_at_build=None, nl=None) -> NeighborList:
    return ctx.nl_build(pos, box, r_cut, skin, excl_pairs, pos_at_build, nl)


def dimos_nl_needs_rebuild_static(ctx: Context, pos, pos_at_build, skin, flag, max_disp2=None):
    return ctx.nl_needs_rebuild_static(pos, pos_at_build, skin, flag, max_disp2)


def dimos_nl_needs_rebuild(ctx: Context, pos, pos_at_build, skin, sync: bool = True, flag=None):
    """flag: int32 device tensor of one element to receive the result (default: one shared by the context's calls)."""
    return ctx.nl_needs_rebuild(pos, pos_at_build, skin, sync, flag)


def dimos_nonbonded(ctx: Context, nl: NeighborList, pos, charge, type_, lj_table, **kw):
    return ctx.nonbonded(nl, pos, charge, type_, lj_table, **kw)


def dimos_pme_recip(ctx: Context, pos, charge, box, alpha, mesh, **kw):
    return ctx.pme_recip(pos, charge, box, alpha, mesh, **kw)


def dimos_pme_mesh_size(alpha, box, delta):
    """The paper's mesh heuristic, rounded up to 7-smooth sizes: tuple of 3 ints.  Host only."""
    m = (ctypes.c_int32 * 3)()
    rc = load_library().dimos_pme_mesh_size(float(alpha), _box3(box), float(delta), m)
    if rc != 0:
        raise DimosError(rc, "dimos_pme_mesh_size: bad argument")
    return tuple(int(k) for k in m)


def dimos_dispersion_correction(ctx: Context, type_, lj_table, box, r_cut, r_switch=0.0):
    return ctx.dispersion_correction(type_, lj_table, box, r_cut, r_switch)


def dimos_virtual_box(ctx: Context, pos, r_cut, skin):
    return ctx.virtual_box(pos, r_cut, skin)


def dimos_vv_kick_drift(ctx: Context, pos, vel, F, inv_mass, dt, **kw):
    return ctx.vv_kick_drift(pos, vel, F, inv_mass, dt, **kw)


def dimos_vv_kick(ctx: Context, vel, F, inv_mass, dt, skip_flag=None):
    return ctx.vv_kick(vel, F, inv_mass, dt, skip_flag)


def dimos_langevin_ou(ctx: Context, vel, inv_mass, xi, gamma, dt, T):
    return ctx.langevin_ou(vel, inv_mass, xi, gamma, dt, T)


def dimos_settle(ctx: Context, pos_old, pos, water, m_O, m_H, d_OH, d_HH, vel=None, dt=0.0):
    return ctx.settle(pos_old, pos, water, m_O, m_H, d_OH, d_HH, vel=vel, dt=dt)


def dimos_settle_velocities(ctx: Context, pos, vel, water, m_O, m_H):
    return ctx.settle_velocities(pos, vel, water, m_O, m_H)


def dimos_water_kick_drift_settle(ctx: Context, pos, vel, F, water, m_O, m_H, d_OH, d_HH, dt, **kw):
    return ctx.water_kick_drift_settle(pos, vel, F, water, m_O, m_H, d_OH, d_HH, dt, **kw)


def dimos_water_kick_settle_velocities(ctx: Context, pos, vel, F, water, m_O, m_H, dt, want_ke=False, skip_flag=None):
    return ctx.water_kick_settle_velocities(pos, vel, F, water, m_O, m_H, dt, want_ke=want_ke, skip_flag=skip_flag)


def dimos_berendsen_scale(ctx: Context, vel, n_dof, T0, tau, dt, ke):
    return ctx.berendsen_scale(vel, n_dof, T0, tau, dt, ke)


def dimos_kinetic_energy(ctx: Context, vel, inv_mass):
    return ctx.kinetic_energy(vel, inv_mass)


def dimos_berendsen(ctx: Context, vel, inv_mass, n_dof, T0, tau, dt, sync=True):
    return ctx.berendsen(vel, inv_mass, n_dof, T0, tau, dt, sync=sync)


def dimos_nl_set_exceptions(ctx: Context, nl: NeighborList, pairs, scale):
    return ctx.nl_set_exceptions(nl, pairs, scale)


def dimos_nl_export_edges(ctx: Context, nl: NeighborList, radius: float):
    return ctx.nl_export_edges(nl, radius)


def dimos_nl_export_pairs(ctx: Context, nl: NeighborList) -> torch.Tensor:
    return ctx.nl_export_pairs(nl)


def lj_table_from_types(sigma, epsilon) -> torch.Tensor:
    """Host-side fill of the (sigma_ab, eps_ab) table by Lorentz-Berthelot, Eq. (5) PAPER.md:195."""
    s = torch.as_tensor(sigma, dtype=torch.float64).contiguous()
    e = torch.as_tensor(epsilon, dtype=torch.float64).contiguous()
    table = torch.empty(s.numel(), s.numel(), 2, dtype=torch.float64)
    rc = load_library().dimos_lj_table_fill(s.data_ptr(), e.data_ptr(), s.numel(), table.data_ptr())  # dimos_lj_table_fill
    if rc != 0:
        raise DimosError(rc, "dimos_lj_table_fill: bad argument")
    return table


dimos_lj_table_fill = lj_table_from_types
