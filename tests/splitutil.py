"""Test helper for the local / non-local split: reorder a workload so that its "local" molecules come first.
Pure index bookkeeping (no arithmetic of the method): molecules stay contiguous, exclusions are remapped."""
import dataclasses

import numpy as np


def local_first(w, is_local_atom):
    """Returns (workload with the molecules whose FIRST atom satisfies is_local_atom(x) moved to the front, nlocal).
    is_local_atom maps the [N,3] coordinates to a boolean per atom."""
    n = w.natoms
    mol = w.mol_of_atom
    nmol = int(mol.max()) + 1
    first = np.full(nmol, n, dtype=np.int64)
    np.minimum.at(first, mol, np.arange(n))
    flag_mol = is_local_atom(w.x)[first]
    # stable: local molecules in their old order, then the others; atoms of a molecule keep their order
    key = np.where(flag_mol[mol], 0, 1)
    perm = np.argsort(key, kind="stable")          # new position k holds old atom perm[k]
    inv = np.empty(n, dtype=np.int64)
    inv[perm] = np.arange(n)
    nlocal = int((key == 0).sum())
    off = [0]
    idx = []
    for k in range(n):
        o = perm[k]
        row = np.sort(inv[w.excl_idx[w.excl_off[o]:w.excl_off[o + 1]]])
        idx.extend(int(v) for v in row)
        off.append(len(idx))
    new_mol_ids = {}
    mol_new = np.empty(n, dtype=np.int32)
    for k in range(n):
        mol_new[k] = new_mol_ids.setdefault(int(mol[perm[k]]), len(new_mol_ids))
    old_of_new_mol = np.array(sorted(new_mol_ids, key=new_mol_ids.get), dtype=np.int64)
    w2 = dataclasses.replace(
        w, name=w.name + "_localfirst", x=np.ascontiguousarray(w.x[perm]), q=np.ascontiguousarray(w.q[perm]),
        type=np.ascontiguousarray(w.type[perm]), excl_off=np.asarray(off, dtype=np.int32),
        excl_idx=np.asarray(idx, dtype=np.int32), mol_of_atom=mol_new,
        unit_dir=np.ascontiguousarray(w.unit_dir[old_of_new_mol]))
    return w2, nlocal
