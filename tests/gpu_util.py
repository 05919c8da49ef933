"""Helpers for the GPU parity tests: drive the C ABI through the Python binding and run the
oracle on the same seeded inputs."""
import numpy as np

from oracle import oracle as O
from tests import listcheck as LC


def oracle_params(w, **kw):
    beta = O.beta_from_rtol(w.rc, w.ewald_rtol) if w.coulomb == "ewald" else 0.0
    return O.Params(rc=w.rc, ntypes=w.ntypes, coulomb=w.coulomb, beta=beta, **kw)


def oracle_forces(w, x=None, method="allpairs", **kw):
    return O.forces(w.x if x is None else x, w.q, w.type, w.box, w.lj_c6c12, w.excl_off, w.excl_idx,
                    oracle_params(w, **kw), method=method)


class Driver:
    """put_atoms / search / prune / forces on torch tensors for one workload."""

    def __init__(self, w, **ctx_kw):
        import torch
        from paper_2006_09167_b200 import nb
        self.torch, self.nb, self.w = torch, nb, w
        self.dev = torch.device("cuda", 0)
        self.ctx = nb.context_for(w, **ctx_kw)
        self.q = torch.from_numpy(w.q).to(self.dev)
        self.t = torch.from_numpy(w.type).to(self.dev)
        self.f = torch.zeros((w.natoms, 3), dtype=torch.float32, device=self.dev)
        self.e = torch.zeros(2, dtype=torch.float64, device=self.dev)
        self.v = torch.zeros(9, dtype=torch.float64, device=self.dev)

    def put(self, x=None):
        x = self.w.x if x is None else x
        self.x = self.torch.from_numpy(np.ascontiguousarray(x, dtype=np.float32)).to(self.dev)
        self.ctx.put_atoms(self.x, self.q, self.t, self.w.box)

    def forces(self, energy=False, virial=False):
        self.f.fill_(float("nan"))
        self.ctx.forces(self.f, self.e if energy else None, self.v if virial else None)
        self.torch.cuda.synchronize()
        out = [self.f.cpu().numpy().astype(np.float64)]
        if energy:
            out.append(self.e.cpu().numpy().copy())
        if virial:
            out.append(self.v.cpu().numpy().reshape(3, 3).copy())
        return out[0] if len(out) == 1 else tuple(out)

    def slots(self):
        aos, xq = self.ctx.get_slots()
        return aos.cpu().numpy(), xq.cpu().numpy()

    def dump(self, which):
        ci, cj, sid, pm, part = self.ctx.list_dump(which)
        return ci, cj, self.nb.shift_vectors(sid), pm, part

    def inner_dump(self):
        """The compact half-cluster inner list: ci, entry, shift vectors, kind, part."""
        ci, ent, sid, kind, part = self.ctx.inner_dump()
        return ci, ent, self.nb.shift_vectors(sid), kind, part


def rel_rms(f, ref):
    return float(np.sqrt(((f - ref) ** 2).sum() / (ref**2).sum()))
