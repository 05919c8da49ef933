"""Thin Python binding of the C ABI in include/nb.h (argument marshalling only).

Every step of the path runs in the CUDA kernels behind libnb_b200.so; PyTorch is used for
device memory and streams.  There is no CPU fallback: if the library has not been built
(`python -m paper_2006_09167_b200.build`) importing this module's functions raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libnb_b200.so")

NB_OK = 0
NB_ERR = {-1: "NB_ERR_ARG", -2: "NB_ERR_STATE", -3: "NB_ERR_CUTOFF", -4: "NB_ERR_BOX", -5: "NB_ERR_NOMEM",
          -6: "NB_ERR_CUDA", -7: "NB_ERR_OVERFLOW"}
NB_COUL_EWALD, NB_COUL_RF, NB_COUL_NONE = 0, 1, 2
NB_MOD_NONE, NB_MOD_POTSHIFT = 0, 1
NB_SHIFT_CENTER = 13

EXPORTS = ["nb_init", "nb_put_atoms", "nb_put_atoms_host", "nb_search", "nb_prune", "nb_forces",
           "nb_forces_host", "nb_free", "nb_last_error", "nb_get_layout", "nb_get_slots", "nb_list_count",
           "nb_list_dump", "nb_get_stats", "nb_measure_fp32_peak", "nb_count_pairs", "nb_timing_enable",
           "nb_timing_read", "nb_timing_stages", "nb_count_slots", "nb_inner_dump", "nb_prune_overlapped", "nb_forces_prune", "nb_step", "nb_measure_fp32_pipe", "nb_step_host",
           "nb_forces_static", "nb_set_local", "nb_forces_nonlocal", "nb_forces_local", "nb_sync_nonlocal", "nb_split_info"]
NB_T_NAMES = ["put", "grid", "search", "masks", "prune", "force", "reduce", "force_energy"]


class nb_params(C.Structure):
    _fields_ = [("natoms", C.c_int32), ("ntypes", C.c_int32), ("lj_c6c12", C.c_void_p),
                ("excl_off", C.c_void_p), ("excl_idx", C.c_void_p), ("rc", C.c_float),
                ("coulomb", C.c_int32), ("ewald_beta", C.c_float), ("ewald_rtol", C.c_float),
                ("eps_rf", C.c_float), ("epsfac", C.c_float), ("lj_modifier", C.c_int32),
                ("coul_modifier", C.c_int32), ("device", C.c_int32), ("stream", C.c_void_p), ("rc_vdw", C.c_float)]


class nb_stats(C.Structure):
    _fields_ = [("cluster_size", C.c_int32), ("nclusters", C.c_int32), ("nsuper", C.c_int32),
                ("nslots", C.c_int32), ("ncolumns_x", C.c_int32), ("ncolumns_y", C.c_int32),
                ("n_sci_entries", C.c_int64), ("n_joint_outer", C.c_int64), ("n_pairs_outer", C.c_int64),
                ("n_pairs_inner", C.c_int64), ("n_excl_masks", C.c_int64), ("n_work_units", C.c_int64),
                ("slots_last_forces", C.c_int64), ("kernel_launches", C.c_int64), ("search_count", C.c_int64),
                ("prune_count", C.c_int64), ("force_count", C.c_int64), ("list_grow_retries", C.c_int32),
                ("ewald_beta", C.c_float)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


_lib = None


def lib():
    """Loads libnb_b200.so; raises if it is missing (no fallback of any kind)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2006_09167_b200.build` "
                               "(there is no CPU or PyTorch fallback for the non-bonded path)")
        _lib = C.CDLL(LIB_PATH)
        _lib.nb_last_error.restype = C.c_char_p
        _lib.nb_free.restype = None
    return _lib


class NbError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"{NB_ERR.get(code, code)}: {msg}")
        self.code = code


def _dptr(t):
    return C.c_void_p(t.data_ptr()) if t is not None else C.c_void_p(0)


def _hptr(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else C.c_void_p(0)


class Context:
    """One nb_ctx.  Methods carry the names of the ABI calls they marshal for."""

    def __init__(self, natoms, lj_c6c12, excl_off, excl_idx, rc, coulomb="ewald", ewald_beta=0.0,
                 ewald_rtol=1e-5, eps_rf=0.0, epsfac=0.0, lj_modifier=NB_MOD_POTSHIFT,
                 coul_modifier=NB_MOD_POTSHIFT, device=0, stream=None, rc_vdw=0.0):
        import torch
        self._torch = torch
        self.natoms = int(natoms)
        lj = np.ascontiguousarray(lj_c6c12, dtype=np.float32)
        self.ntypes = int(round((lj.size // 2) ** 0.5))
        eo = np.ascontiguousarray(excl_off, dtype=np.int32) if excl_off is not None else None
        ei = np.ascontiguousarray(excl_idx, dtype=np.int32) if excl_idx is not None else None
        if ei is not None and ei.size == 0:
            ei = np.zeros(1, dtype=np.int32)
        self.device = torch.device("cuda", device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        p = nb_params(self.natoms, self.ntypes, _hptr(lj), _hptr(eo), _hptr(ei), float(rc),
                      {"ewald": NB_COUL_EWALD, "rf": NB_COUL_RF, "none": NB_COUL_NONE}[coulomb], float(ewald_beta), float(ewald_rtol),
                      float(eps_rf), float(epsfac), int(lj_modifier), int(coul_modifier), int(device),
                      C.c_void_p(self.stream.cuda_stream), float(rc_vdw))
        self._h = C.c_void_p(0)
        rcode = lib().nb_init(C.byref(p), C.byref(self._h))
        if rcode != NB_OK:
            msg = lib().nb_last_error(self._h).decode() if self._h else "nb_init failed"
            if self._h:
                lib().nb_free(self._h)
                self._h = C.c_void_p(0)
            raise NbError(rcode, msg)

    def _check(self, rcode):
        if rcode != NB_OK:
            raise NbError(rcode, lib().nb_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None):
            lib().nb_free(self._h)
            self._h = C.c_void_p(0)

    __del__ = close

    # ---- the five working calls ----
    def put_atoms(self, x, q, typ, box):
        """x [N,3] f32, q [N] f32, typ [N] i32: CUDA tensors; box: 3 floats (host)."""
        b = (C.c_float * 3)(*[float(v) for v in box])
        self._check(lib().nb_put_atoms(self._h, _dptr(x), _dptr(q), _dptr(typ), b))

    def put_atoms_host(self, x, q, typ, box):
        """Same with host numpy arrays (or pinned CPU tensors via .numpy())."""
        b = (C.c_float * 3)(*[float(v) for v in box])
        self._check(lib().nb_put_atoms_host(self._h, _hptr(x), _hptr(q), _hptr(typ), b))

    def search(self, rlist_outer):
        self._check(lib().nb_search(self._h, C.c_float(rlist_outer)))

    def prune(self, rlist_inner, part=0, nparts=1):
        self._check(lib().nb_prune(self._h, C.c_float(rlist_inner), C.c_int(part), C.c_int(nparts)))

    def prune_overlapped(self, rlist_inner, part=0, nparts=1):
        self._check(lib().nb_prune_overlapped(self._h, C.c_float(rlist_inner), C.c_int(part), C.c_int(nparts)))

    def forces(self, f, energies=None, virial=None):
        """f [N,3] f32 CUDA tensor (overwritten); energies [2] f64, virial [9] f64 CUDA tensors or None."""
        self._check(lib().nb_forces(self._h, _dptr(f), _dptr(energies), _dptr(virial)))

    def set_local(self, nlocal):
        """Atoms [0, nlocal) are local, the rest non-local (halo); takes effect at the next search."""
        self._check(lib().nb_set_local(self._h, C.c_int32(int(nlocal))))

    def forces_nonlocal(self, f, energies=None, virial=None):
        self._check(lib().nb_forces_nonlocal(self._h, _dptr(f), _dptr(energies), _dptr(virial)))

    def forces_local(self, f):
        self._check(lib().nb_forces_local(self._h, _dptr(f)))

    def sync_nonlocal(self):
        self._check(lib().nb_sync_nonlocal(self._h))

    def split_info(self):
        v = [C.c_int32() for _ in range(4)]
        self._check(lib().nb_split_info(self._h, *[C.byref(a) for a in v]))
        return dict(nlocal=v[0].value, nclusters_local=v[1].value, nseg_local=v[2].value, nseg=v[3].value)

    def forces_static(self, f, energies=None, virial=None):
        """nb_forces without any allocation: the kernel's scratch is a static device array of the library (size limit:
        nb.h NB_STATIC_MAX_SLOTS; calls that overlap on the GPU race)."""
        self._check(lib().nb_forces_static(self._h, _dptr(f), _dptr(energies), _dptr(virial)))

    def step(self, x, rlist_inner, part, nparts, f):
        self._check(lib().nb_step(self._h, _dptr(x), C.c_float(rlist_inner), C.c_int(part), C.c_int(nparts), _dptr(f)))

    def step_host(self, x, f, rlist_inner, part, nparts):
        self._check(lib().nb_step_host(self._h, _hptr(x), _hptr(f), C.c_float(rlist_inner), C.c_int(part), C.c_int(nparts)))

    def forces_prune(self, rlist_inner, f, energies=None, virial=None):
        """The fused first prune: forces over the outer list + the whole inner list for rlist_inner in one kernel."""
        self._check(lib().nb_forces_prune(self._h, C.c_float(rlist_inner), _dptr(f), _dptr(energies), _dptr(virial)))

    def forces_host(self, f, energies=None, virial=None):
        self._check(lib().nb_forces_host(self._h, _hptr(f), _hptr(energies), _hptr(virial)))

    # ---- introspection ----
    def get_layout(self):
        v = [C.c_int32() for _ in range(4)]
        self._check(lib().nb_get_layout(self._h, *[C.byref(a) for a in v]))
        return dict(cluster_size=v[0].value, nclusters=v[1].value, nsuper=v[2].value, nslots=v[3].value)

    def get_slots(self):
        torch = self._torch
        n = self.get_layout()["nslots"]
        aos = torch.empty(n, dtype=torch.int32, device=self.device)
        xq = torch.empty((n, 4), dtype=torch.float32, device=self.device)
        self._check(lib().nb_get_slots(self._h, _dptr(aos), _dptr(xq)))
        return aos, xq

    def list_count(self, which):
        n = C.c_int64()
        self._check(lib().nb_list_count(self._h, C.c_int(which), C.byref(n)))
        return n.value

    def list_dump(self, which):
        """Returns numpy arrays ci, cj, shift id, pairmask (uint64), part."""
        torch = self._torch
        n = self.list_count(which)
        mk = lambda dt: torch.empty(max(n, 1), dtype=dt, device=self.device)
        ci, cj, sh, part = mk(torch.int32), mk(torch.int32), mk(torch.int32), mk(torch.int32)
        pm = mk(torch.int64)
        self._check(lib().nb_list_dump(self._h, C.c_int(which), _dptr(ci), _dptr(cj), _dptr(sh), _dptr(pm), _dptr(part)))
        out = [t[:n].cpu().numpy() for t in (ci, cj, sh)]
        return out[0], out[1], out[2], pm[:n].cpu().numpy().view(np.uint64), part[:n].cpu().numpy()

    def get_stats(self):
        s = nb_stats()
        self._check(lib().nb_get_stats(self._h, C.byref(s)))
        return s.as_dict()

    def measure_fp32_peak(self):
        v = C.c_double()
        self._check(lib().nb_measure_fp32_peak(self._h, C.byref(v)))
        return v.value


    def measure_fp32_pipe(self):
        v = (C.c_double * 4)()
        self._check(lib().nb_measure_fp32_pipe(self._h, v))
        return {"ffma_3reg": v[0], "ffma2_3pairs": v[1], "ffma2_pair_pair_const": v[2], "fmul2_2pairs": v[3]}

    def count_pairs(self):
        """(interacting, excluded) atom pairs with r < rc over the inner list."""
        a, b = C.c_int64(), C.c_int64()
        self._check(lib().nb_count_pairs(self._h, C.byref(a), C.byref(b)))
        return a.value, b.value

    def count_slots(self):
        """Atom-pair slots the force kernel evaluates over the inner list (raw pair count)."""
        n = C.c_int64()
        self._check(lib().nb_count_slots(self._h, C.byref(n)))
        return n.value

    def inner_dump(self):
        """The compact inner list the force kernel streams: numpy arrays ci, entry, shift id, kind
        (0: entry = slot of a listed j atom; 1: entry = whole j-cluster with a mask), part."""
        n = C.c_int64()
        null = C.c_void_p(0)
        self._check(lib().nb_inner_dump(self._h, C.byref(n), null, null, null, null, null))
        arr = [np.zeros(max(n.value, 1), dtype=np.int32) for _ in range(5)]
        self._check(lib().nb_inner_dump(self._h, C.byref(n), *[_hptr(a) for a in arr]))
        return tuple(a[: n.value] for a in arr)

    def timing_enable(self, on=True):
        self._check(lib().nb_timing_enable(self._h, C.c_int(int(on))))

    def timing_stages(self, mask=0xFFFFFFFF):
        self._check(lib().nb_timing_stages(self._h, C.c_uint(int(mask))))

    def timing_read(self, reset=True):
        """{stage: (milliseconds, intervals)} accumulated since the last reset."""
        ms = (C.c_double * len(NB_T_NAMES))()
        cnt = (C.c_int64 * len(NB_T_NAMES))()
        self._check(lib().nb_timing_read(self._h, ms, cnt, C.c_int(int(reset))))
        return {k: (ms[i], cnt[i]) for i, k in enumerate(NB_T_NAMES)}


def shift_vectors(shift_id):
    """(sx,sy,sz) of ABI shift ids: id = (sx+1) + 3*(sy+1) + 9*(sz+1)."""
    s = np.asarray(shift_id).astype(np.int64)
    return np.stack([s % 3 - 1, (s // 3) % 3 - 1, s // 9 - 1], axis=-1)


def context_for(w, device=0, stream=None, **overrides):
    """Context for a workloads.Workload with the run parameters its config names."""
    kw = dict(rc=w.rc, coulomb=w.coulomb, ewald_rtol=w.ewald_rtol)
    kw.update(overrides)
    return Context(w.natoms, w.lj_c6c12, w.excl_off, w.excl_idx, device=device, stream=stream, **kw)
