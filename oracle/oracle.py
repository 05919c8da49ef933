"""ctypes front-end of oracle/nb_oracle.c (fp64 CPU oracle; test infrastructure only).

Every function promotes the fp32 inputs to fp64 exactly and calls the C routine that
states the definition (see the header of nb_oracle.c for the citations).  Nothing here
imports or calls the CUDA path.
"""
from __future__ import annotations

import ctypes as C
import dataclasses

import numpy as np

from . import build_oracle

_lib = None


class _Params(C.Structure):
    _fields_ = [("coulomb", C.c_int32), ("lj_shift", C.c_int32), ("coul_shift", C.c_int32),
                ("ntypes", C.c_int32), ("rc", C.c_double), ("beta", C.c_double),
                ("eps_rf", C.c_double), ("epsfac", C.c_double), ("rc_vdw", C.c_double)]


EPSFAC = 138.935458  # reading A2


@dataclasses.dataclass
class Params:
    rc: float
    ntypes: int
    coulomb: str = "ewald"  # "ewald" | "rf" | "none" (LJ only)
    beta: float = 0.0
    eps_rf: float = 0.0  # <= 0: infinity
    epsfac: float = EPSFAC
    lj_shift: bool = True
    coul_shift: bool = True
    rc_vdw: float = 0.0  # twin cut-offs: LJ cut-off <= rc; <= 0: same as rc

    def c(self) -> _Params:
        return _Params({"ewald": 0, "rf": 1, "none": 2}[self.coulomb], int(self.lj_shift), int(self.coul_shift),
                       int(self.ntypes), float(self.rc), float(self.beta), float(self.eps_rf),
                       float(self.epsfac), float(self.rc_vdw))


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build_oracle.build())
        _lib.oracle_beta_from_rtol.restype = C.c_double
        _lib.oracle_beta_from_rtol.argtypes = [C.c_double, C.c_double]
        _lib.oracle_lists.restype = C.c_longlong
        _lib.oracle_num_threads.restype = C.c_int
    return _lib


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def beta_from_rtol(rc: float, rtol: float) -> float:
    return float(lib().oracle_beta_from_rtol(float(rc), float(rtol)))


def pair(p: Params, r: float, qq: float, c6: float, c12: float, excluded: bool):
    """(V_lj, V_c, F_lj, F_c) of one pair at distance r (radial forces, -dV/dr)."""
    out = [C.c_double() for _ in range(4)]
    pc = p.c()
    lib().oracle_pair(C.byref(pc), C.c_double(r), C.c_double(qq), C.c_double(c6), C.c_double(c12),
                      C.c_int(int(excluded)), *[C.byref(o) for o in out])
    return tuple(o.value for o in out)


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p)


@dataclasses.dataclass
class ForceResult:
    f: np.ndarray  # float64 [N,3]
    e_lj: float
    e_coul: float
    virial: np.ndarray  # float64 [3,3]
    npairs: int  # non-excluded pairs with r < rc ("effective" pairs)
    npairs_excl: int

    @property
    def energy(self) -> float:
        return self.e_lj + self.e_coul


def forces(x, q, typ, box, lj_c6c12, excl_off, excl_idx, p: Params, method: str = "allpairs") -> ForceResult:
    """method: 'allpairs' (the definition), 'cells' (same sum, linked cells), 'images' (T5 brute force)."""
    x64 = np.ascontiguousarray(x, dtype=np.float64)
    q64 = np.ascontiguousarray(q, dtype=np.float64)
    t = np.ascontiguousarray(typ, dtype=np.int32)
    b64 = np.ascontiguousarray(box, dtype=np.float64)
    lj = np.ascontiguousarray(lj_c6c12, dtype=np.float32)
    eo = np.ascontiguousarray(excl_off, dtype=np.int32)
    ei = np.ascontiguousarray(excl_idx, dtype=np.int32)
    if ei.size == 0:
        ei = np.zeros(1, dtype=np.int32)
    n = x64.shape[0]
    f = np.zeros((n, 3), dtype=np.float64)
    e = np.zeros(2, dtype=np.float64)
    vir = np.zeros(9, dtype=np.float64)
    npairs = np.zeros(2, dtype=np.int64)
    fn = {"allpairs": lib().oracle_forces_allpairs, "cells": lib().oracle_forces_cells,
          "images": lib().oracle_forces_images}[method]
    pc = p.c()
    rcode = fn(C.c_int(n), _ptr(x64), _ptr(q64), _ptr(t), _ptr(b64), _ptr(lj), _ptr(eo), _ptr(ei),
               C.byref(pc), _ptr(f), _ptr(e), _ptr(vir), _ptr(npairs))
    if rcode != 0:
        raise RuntimeError(f"oracle {method} refused the box (fewer than 3 cells per axis)")
    return ForceResult(f, float(e[0]), float(e[1]), vir.reshape(3, 3), int(npairs[0]), int(npairs[1]))


def forces_split(x, q, typ, box, lj_c6c12, excl_off, excl_idx, p: Params, nlocal: int, which: int) -> ForceResult:
    """Local / non-local split (reading A25): which = 1 pairs among the local atoms [0, nlocal),
    which = 2 pairs with at least one non-local atom, which = 0 all pairs."""
    x64 = np.ascontiguousarray(x, dtype=np.float64)
    q64 = np.ascontiguousarray(q, dtype=np.float64)
    t = np.ascontiguousarray(typ, dtype=np.int32)
    b64 = np.ascontiguousarray(box, dtype=np.float64)
    lj = np.ascontiguousarray(lj_c6c12, dtype=np.float32)
    eo = np.ascontiguousarray(excl_off, dtype=np.int32)
    ei = np.ascontiguousarray(excl_idx, dtype=np.int32)
    if ei.size == 0:
        ei = np.zeros(1, dtype=np.int32)
    n = x64.shape[0]
    f = np.zeros((n, 3), dtype=np.float64)
    e = np.zeros(2, dtype=np.float64)
    vir = np.zeros(9, dtype=np.float64)
    npairs = np.zeros(2, dtype=np.int64)
    pc = p.c()
    lib().oracle_forces_split(C.c_int(n), C.c_int(int(nlocal)), C.c_int(int(which)), _ptr(x64), _ptr(q64), _ptr(t),
                              _ptr(b64), _ptr(lj), _ptr(eo), _ptr(ei), C.byref(pc), _ptr(f), _ptr(e), _ptr(vir),
                              _ptr(npairs))
    return ForceResult(f, float(e[0]), float(e[1]), vir.reshape(3, 3), int(npairs[0]), int(npairs[1]))


def virial_shift_identity(x, q, typ, box, lj_c6c12, excl_off, excl_idx, p: Params) -> np.ndarray:
    x64 = np.ascontiguousarray(x, dtype=np.float64)
    q64 = np.ascontiguousarray(q, dtype=np.float64)
    t = np.ascontiguousarray(typ, dtype=np.int32)
    b64 = np.ascontiguousarray(box, dtype=np.float64)
    lj = np.ascontiguousarray(lj_c6c12, dtype=np.float32)
    eo = np.ascontiguousarray(excl_off, dtype=np.int32)
    ei = np.ascontiguousarray(excl_idx, dtype=np.int32)
    if ei.size == 0:
        ei = np.zeros(1, dtype=np.int32)
    vir = np.zeros(9, dtype=np.float64)
    pc = p.c()
    lib().oracle_virial_shift_identity(C.c_int(x64.shape[0]), _ptr(x64), _ptr(q64), _ptr(t), _ptr(b64),
                                       _ptr(lj), _ptr(eo), _ptr(ei), C.byref(pc), _ptr(vir))
    return vir.reshape(3, 3)


@dataclasses.dataclass
class ListResult:
    ci: np.ndarray  # int32 [n]
    cj: np.ndarray  # int32 [n]
    s: np.ndarray  # int8 [n,3]  shift of the FIRST cluster: d = x_a + s L - x_b
    inner: np.ndarray  # bool [n]
    pairmask: np.ndarray  # uint64 [n], bit a*C+b

    def keys(self, which: str = "outer") -> np.ndarray:
        """Unique int64 key per canonical triple (for set comparison)."""
        sid = (self.s[:, 0].astype(np.int64) + 1) * 9 + (self.s[:, 1].astype(np.int64) + 1) * 3 \
            + (self.s[:, 2].astype(np.int64) + 1)
        k = (self.ci.astype(np.int64) << 36) | (self.cj.astype(np.int64) << 8) | sid
        return k if which == "outer" else k[self.inner]


def lists(atom_of_slot, xq, box, rlist_outer, rlist_inner, excl_off, excl_idx, cluster_size=8,
          c_begin=0, c_end=None) -> ListResult:
    """Canonical outer triples, inner flags and pairmasks (S:8.3.2) on the exported layout."""
    aos = np.ascontiguousarray(atom_of_slot, dtype=np.int32)
    xq32 = np.ascontiguousarray(xq, dtype=np.float32).reshape(-1, 4)
    b32 = np.ascontiguousarray(box, dtype=np.float32)
    eo = np.ascontiguousarray(excl_off, dtype=np.int32)
    ei = np.ascontiguousarray(excl_idx, dtype=np.int32)
    if ei.size == 0:
        ei = np.zeros(1, dtype=np.int32)
    ncl = aos.shape[0] // cluster_size
    if c_end is None:
        c_end = ncl
    cap = 0
    bufs = None
    for _ in range(2):
        ci = np.zeros(max(cap, 1), dtype=np.int32)
        cj = np.zeros(max(cap, 1), dtype=np.int32)
        s = np.zeros((max(cap, 1), 3), dtype=np.int8)
        inner = np.zeros(max(cap, 1), dtype=np.uint8)
        mask = np.zeros(max(cap, 1), dtype=np.uint64)
        n = lib().oracle_lists(C.c_int(ncl), C.c_int(cluster_size), _ptr(aos), _ptr(xq32), _ptr(b32),
                               C.c_float(rlist_outer), C.c_float(rlist_inner), _ptr(eo), _ptr(ei),
                               C.c_int(c_begin), C.c_int(c_end), C.c_longlong(cap), _ptr(ci), _ptr(cj),
                               _ptr(s), _ptr(inner), _ptr(mask))
        if n <= cap:
            bufs = (ci[:n], cj[:n], s[:n], inner[:n].astype(bool), mask[:n])
            break
        cap = int(n)
    return ListResult(*bufs)


@dataclasses.dataclass
class HalfListResult:
    ci: np.ndarray  # int32 [n]
    entry: np.ndarray  # int32 [n]   kind 0: 2*cj + half;  kind 1: cj
    s: np.ndarray  # int8 [n,3]   shift of ci, as in ListResult
    kind: np.ndarray  # uint8 [n]  0 = half j-cluster of a cluster pair with a trivial mask, 1 = whole masked cluster pair

    def keys(self) -> np.ndarray:
        """Unique int64 key per entry (ci, entry, shift, kind)."""
        sid = (self.s[:, 0].astype(np.int64) + 1) * 9 + (self.s[:, 1].astype(np.int64) + 1) * 3 \
            + (self.s[:, 2].astype(np.int64) + 1)
        return (self.ci.astype(np.int64) << 38) | (self.entry.astype(np.int64) << 9) | (sid << 1) | self.kind.astype(np.int64)


def half_lists(atom_of_slot, xq, box, rlist_outer, rlist_inner, excl_off, excl_idx, cluster_size=8,
               c_begin=0, c_end=None, fn="oracle_half_lists") -> HalfListResult:
    """The inner list at half-j-cluster granularity (oracle_half_lists) on the exported layout."""
    aos = np.ascontiguousarray(atom_of_slot, dtype=np.int32)
    xq32 = np.ascontiguousarray(xq, dtype=np.float32).reshape(-1, 4)
    b32 = np.ascontiguousarray(box, dtype=np.float32)
    eo = np.ascontiguousarray(excl_off, dtype=np.int32)
    ei = np.ascontiguousarray(excl_idx, dtype=np.int32)
    if ei.size == 0:
        ei = np.zeros(1, dtype=np.int32)
    ncl = aos.shape[0] // cluster_size
    if c_end is None:
        c_end = ncl
    getattr(lib(), fn).restype = C.c_longlong
    cap = 0
    for _ in range(2):
        ci = np.zeros(max(cap, 1), dtype=np.int32)
        ent = np.zeros(max(cap, 1), dtype=np.int32)
        s = np.zeros((max(cap, 1), 3), dtype=np.int8)
        kind = np.zeros(max(cap, 1), dtype=np.uint8)
        n = getattr(lib(), fn)(C.c_int(ncl), C.c_int(cluster_size), _ptr(aos), _ptr(xq32), _ptr(b32),
                                    C.c_float(rlist_outer), C.c_float(rlist_inner), _ptr(eo), _ptr(ei),
                                    C.c_int(c_begin), C.c_int(c_end), C.c_longlong(cap), _ptr(ci), _ptr(ent),
                                    _ptr(s), _ptr(kind))
        if n <= cap:
            return HalfListResult(ci[:n], ent[:n], s[:n], kind[:n])
        cap = int(n)
    raise RuntimeError("oracle_half_lists: count changed between passes")


def atom_lists(atom_of_slot, xq, box, rlist_outer, rlist_inner, excl_off, excl_idx, cluster_size=8, c_begin=0, c_end=None):
    """The inner list at single-j-ATOM granularity (oracle_atom_lists): kind-0 entries are j slot indices."""
    return half_lists(atom_of_slot, xq, box, rlist_outer, rlist_inner, excl_off, excl_idx, cluster_size, c_begin, c_end,
                      fn="oracle_atom_lists")
