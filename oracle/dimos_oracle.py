"""ctypes wrapper around oracle/dimos_oracle.c (argument marshalling only; all arithmetic is in C).

TEST INFRASTRUCTURE ONLY -- see the header of dimos_oracle.c.  Inputs are promoted to float64
here, so an fp32 test input enters the oracle as the same real numbers the GPU path reads.
"""
from __future__ import annotations

import ctypes
import dataclasses

import numpy as np

from . import build_oracle

METHOD_RF = 0
METHOD_EWALD_REAL = 1


class _Params(ctypes.Structure):
    _fields_ = [
        ("r_cut", ctypes.c_double),
        ("eps_rf", ctypes.c_double),
        ("alpha", ctypes.c_double),
        ("coulomb_const", ctypes.c_double),
        ("method", ctypes.c_int32),
        ("r_switch", ctypes.c_double),
    ]


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build_oracle.build())
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int32)
        i64 = ctypes.c_int64
        nb_args = [i64, dp, dp, ip, dp, ctypes.c_int32, dp, ctypes.POINTER(_Params), ip, i64, ctypes.c_double,
                   dp, dp, dp, dp, ctypes.POINTER(i64)]
        for name in ("orc_nonbonded_bruteforce", "orc_nonbonded_celllist"):
            fn = getattr(lib, name)
            fn.argtypes = nb_args
            fn.restype = ctypes.c_int
        for name in ("orc_neighbor_pairs_bruteforce", "orc_neighbor_pairs_celllist"):
            fn = getattr(lib, name)
            fn.argtypes = [i64, dp, dp, ctypes.c_double, ip, i64, ip, i64]
            fn.restype = i64
        lib.orc_add_exceptions.argtypes = [i64, dp, dp, ip, dp, ctypes.c_int32, dp, ctypes.c_double, ip, dp, i64, dp, dp, dp]
        lib.orc_add_exceptions.restype = ctypes.c_int
        lib.orc_needs_rebuild.argtypes = [i64, dp, dp, ctypes.c_double, dp]
        lib.orc_needs_rebuild.restype = ctypes.c_int
        lib.orc_lorentz_berthelot.argtypes = [dp, dp, ctypes.c_int32, dp]
        lib.orc_lorentz_berthelot.restype = None
        lib.orc_num_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def _d(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def _dp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _ip(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_int32))


def num_threads() -> int:
    return int(_load().orc_num_threads())


def lorentz_berthelot(sigma, epsilon) -> np.ndarray:
    """Eq. (5), PAPER.md:195 -> table (ntypes, ntypes, 2) = (sigma_ab, eps_ab)."""
    sigma, epsilon = _d(sigma), _d(epsilon)
    nt = sigma.shape[0]
    table = np.zeros((nt, nt, 2), dtype=np.float64)
    _load().orc_lorentz_berthelot(_dp(sigma), _dp(epsilon), nt, _dp(table))
    return table


@dataclasses.dataclass
class NonbondedResult:
    F: np.ndarray  # (N,3) float64
    E: np.ndarray  # (4,) total, lj, coul_pair, coul_excl_corr
    W: np.ndarray  # (3,3) virial
    n_pairs: int  # unordered in-cutoff pairs
    allow: np.ndarray | None  # (N,) cutoff-band force allowance (C-10) or None


def nonbonded(pos, charge, type_, lj_table, box, r_cut, *, method=METHOD_RF, eps_rf=78.5, alpha=3.12,
              coulomb_const=138.935456, excl_pairs=None, band=0.0, algorithm="celllist", r_switch=0.0,
              exceptions=None) -> NonbondedResult:
    """Forces, energy components and virial for one configuration.  algorithm: 'bruteforce' | 'celllist'.
    r_switch: LJ switching distance r_s of Eq. 6; 0 = plain truncation at r_cut.
    exceptions: (pairs (n,2) int32 i<j, scale (n,2) float64 = (coulomb scale, LJ scale)) of 1-4 exceptions (PAPER.md:243,
    reading C-21); every exception pair must also be listed in excl_pairs."""
    lib = _load()
    pos, charge, type_, box = _d(pos), _d(charge), _i(type_), _d(box)
    lj_table = _d(lj_table)
    n = pos.shape[0]
    nt = lj_table.shape[0]
    excl = _i(excl_pairs if excl_pairs is not None else np.zeros((0, 2), np.int32)).reshape(-1, 2)
    params = _Params(float(r_cut), float(eps_rf), float(alpha), float(coulomb_const), int(method), float(r_switch))
    F = np.zeros((n, 3), dtype=np.float64)
    E = np.zeros(4, dtype=np.float64)
    W = np.zeros(9, dtype=np.float64)
    allow = np.zeros(n, dtype=np.float64) if band > 0 else None
    npairs = ctypes.c_int64(0)
    fn = {"bruteforce": lib.orc_nonbonded_bruteforce, "celllist": lib.orc_nonbonded_celllist}[algorithm]
    rc = fn(n, _dp(pos), _dp(charge), _ip(type_), _dp(lj_table), nt, _dp(box), ctypes.byref(params),
            _ip(excl), excl.shape[0], float(band), _dp(F), _dp(E), _dp(W),
            _dp(allow) if allow is not None else None, ctypes.byref(npairs))
    if rc != 0:
        raise MemoryError(f"oracle nonbonded failed rc={rc}")
    if exceptions is not None:
        ep = _i(exceptions[0]).reshape(-1, 2)
        es = _d(exceptions[1]).reshape(-1, 2)
        if ep.shape[0] != es.shape[0]:
            raise ValueError("exceptions: pairs and scales differ in length")
        have = set(map(tuple, excl.tolist()))
        if any(tuple(p) not in have for p in ep.tolist()):
            raise ValueError("every exception pair must also be an excluded pair")
        lib.orc_add_exceptions(n, _dp(pos), _dp(charge), _ip(type_), _dp(lj_table), nt, _dp(box), float(coulomb_const),
                               _ip(ep), _dp(es), ep.shape[0], _dp(F), _dp(E), _dp(W))
    return NonbondedResult(F, E, W.reshape(3, 3), int(npairs.value), allow)


def neighbor_pairs(pos, box, r_list, excl_pairs=None, algorithm="celllist") -> np.ndarray:
    """Sorted (n,2) int32 array of pairs i<j, not excluded, min-image r < r_list."""
    lib = _load()
    pos, box = _d(pos), _d(box)
    n = pos.shape[0]
    excl = _i(excl_pairs if excl_pairs is not None else np.zeros((0, 2), np.int32)).reshape(-1, 2)
    fn = {"bruteforce": lib.orc_neighbor_pairs_bruteforce, "celllist": lib.orc_neighbor_pairs_celllist}[algorithm]
    total = fn(n, _dp(pos), _dp(box), float(r_list), _ip(excl), excl.shape[0], None, 0)
    if total < 0:
        raise MemoryError(f"oracle neighbor_pairs count failed rc={total}")
    pairs = np.zeros((total, 2), dtype=np.int32)
    got = fn(n, _dp(pos), _dp(box), float(r_list), _ip(excl), excl.shape[0], _ip(pairs), total)
    if got != total:
        raise RuntimeError(f"oracle neighbor_pairs fill failed rc={got}")
    return pairs


def count_pairs(pos, box, r_list, excl_pairs=None, algorithm="celllist") -> int:
    """Number of pairs neighbor_pairs would return (the C routine's count-only call)."""
    lib = _load()
    pos, box = _d(pos), _d(box)
    excl = _i(excl_pairs if excl_pairs is not None else np.zeros((0, 2), np.int32)).reshape(-1, 2)
    fn = {"bruteforce": lib.orc_neighbor_pairs_bruteforce, "celllist": lib.orc_neighbor_pairs_celllist}[algorithm]
    total = fn(pos.shape[0], _dp(pos), _dp(box), float(r_list), _ip(excl), excl.shape[0], None, 0)
    if total < 0:
        raise MemoryError(f"oracle count_pairs failed rc={total}")
    return int(total)


def needs_rebuild(pos, pos_at_build, skin):
    """(flag, max displacement): PAPER.md:175, strict max |dr| > skin/2 on raw coordinates."""
    pos, ref = _d(pos), _d(pos_at_build)
    m = ctypes.c_double(0.0)
    flag = _load().orc_needs_rebuild(pos.shape[0], _dp(pos), _dp(ref), float(skin), ctypes.byref(m))
    return bool(flag), float(m.value)


def edge_vectors(pos, box, pairs):
    """Distance vectors and periodic shifts of an edge list (minimum image, reading C-3): for every
    pair (a, b): shift = nearbyint((r_a - r_b) / L) per axis and d = r_a - r_b - shift * L.  numpy fp64."""
    pos, box = _d(pos), _d(box)
    pairs = np.asarray(pairs, dtype=np.int64).reshape(-1, 2)
    diff = pos[pairs[:, 0]] - pos[pairs[:, 1]]
    shift = np.rint(diff / box)
    return diff - shift * box, shift.astype(np.int64)
