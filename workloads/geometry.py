"""Seeded synthetic geometries and CSR neighbour lists.

Stand-ins for the paper's workloads (water boxes at 1 g/cm^3 ~ 0.100 atoms/A^3,
25-100 atom gas-phase molecules; PAPER.md:81 r_max = 6 A).  No item of any dataset is
reproduced: everything is drawn from workloads.rng.  Holds none of the method's arithmetic.

Edge convention (reading A7): directed edges, both directions present, CSR by centre atom i,
neighbours j ascending within a row, r_e = x_j - x_i + shift (minimum image), edge iff
0 < |r_e| < r_c.  rev[e] = index of the reverse edge (reading A17).
"""
import numpy as np
from scipy.spatial import cKDTree

from . import rng

SPECIES = ("H", "C", "N", "O")
SPECIES_CDF = np.cumsum([0.5, 0.3, 0.1, 0.1])


def periodic_box(seed, n_atoms, box, min_dist=0.9):
    """Random sequential addition: candidate k = uniform point (counters 3k..3k+2 of the
    'positions' stream); accepted iff no accepted atom is closer than min_dist (minimum image)."""
    st = rng.STREAMS["positions"]
    ncell = max(1, int(np.floor(box / min_dist)))
    cs = box / ncell
    cells = {}
    pos = np.empty((n_atoms, 3))
    count = 0
    k = 0
    batch = 4096
    md2 = min_dist * min_dist
    while count < n_atoms:
        idx = np.arange(3 * k, 3 * (k + batch), dtype=np.uint64)
        cand = rng.uniform(seed, st, idx).reshape(batch, 3) * box
        cidx = np.minimum((cand / cs).astype(np.int64), ncell - 1)
        for b in range(batch):
            p = cand[b]
            cx, cy, cz = cidx[b]
            ok = True
            for dx in (-1, 0, 1):
                for dy in (-1, 0, 1):
                    for dz in (-1, 0, 1):
                        lst = cells.get(((cx + dx) % ncell, (cy + dy) % ncell, (cz + dz) % ncell))
                        if not lst:
                            continue
                        for a in lst:
                            d = pos[a] - p
                            d -= box * np.round(d / box)
                            if d[0] * d[0] + d[1] * d[1] + d[2] * d[2] < md2:
                                ok = False
                                break
                        if not ok:
                            break
                    if not ok:
                        break
                if not ok:
                    break
            if ok:
                pos[count] = p
                cells.setdefault((cx, cy, cz), []).append(count)
                count += 1
                if count == n_atoms:
                    break
        k += batch
    if ncell < 3:  # tiny boxes: the 27-cell stencil wraps onto itself, which only repeats checks
        pass
    return pos


def species(seed, n_atoms):
    """H/C/N/O drawn 50/30/10/10 % (reading A21; not used by the hot path)."""
    u = rng.uniform(seed, rng.STREAMS["species"], np.arange(n_atoms))
    return np.searchsorted(SPECIES_CDF, u, side="right").astype(np.int32)


def _csr_from_pairs(n_atoms, i, j, rvec):
    order = np.lexsort((j, i))
    i, j, rvec = i[order], j[order], rvec[order]
    row_ptr = np.zeros(n_atoms + 1, dtype=np.int64)
    np.add.at(row_ptr, i + 1, 1)
    row_ptr = np.cumsum(row_ptr)
    key = i.astype(np.int64) * n_atoms + j
    rev = np.searchsorted(key, j.astype(np.int64) * n_atoms + i)
    assert np.all(key[rev] == j.astype(np.int64) * n_atoms + i), "neighbour list is not symmetric"
    return dict(row_ptr=row_ptr.astype(np.int32), col=j.astype(np.int32), centre=i.astype(np.int32),
                rev=rev.astype(np.int32), rvec=np.ascontiguousarray(rvec))


def neighbour_list_periodic(pos, box, rc):
    assert rc < box / 2, "minimum image needs r_c < L/2 (reading A7)"
    tree = cKDTree(pos, boxsize=box)
    pairs = tree.query_pairs(rc, output_type="ndarray")
    a, b = pairs[:, 0], pairs[:, 1]
    d = pos[b] - pos[a]
    d -= box * np.round(d / box)
    r = np.sqrt((d * d).sum(1))
    keep = (r > 0) & (r < rc)
    a, b, d = a[keep], b[keep], d[keep]
    i = np.concatenate([a, b])
    j = np.concatenate([b, a])
    rvec = np.concatenate([d, -d])
    return _csr_from_pairs(pos.shape[0], i, j, rvec)


def neighbour_list_periodic_typed(pos, box, species, rc_table):
    """Per-edge-type cutoffs: the pair (i, j) is an edge iff 0 < |r| < rc_table[species[i], species[j]] (symmetric
    table).  Built from the plain list at the largest cutoff by dropping the edges beyond their own cutoff -> the same dict plus
    rc_edge[E], the cutoff of every edge."""
    rc_table = np.asarray(rc_table, dtype=np.float64)
    full = neighbour_list_periodic(pos, box, float(rc_table.max()))
    i, j, d = full["centre"].astype(np.int64), full["col"].astype(np.int64), full["rvec"]
    r = np.sqrt((d * d).sum(1))
    rce = rc_table[species[i], species[j]]
    keep = r < rce
    out = _csr_from_pairs(pos.shape[0], i[keep], j[keep], d[keep])
    out["rc_edge"] = rc_table[species[out["centre"]], species[out["col"]]]
    return out


def neighbour_list_open(pos, rc, mol_ptr=None):
    """Non-periodic; with mol_ptr, no edges between different molecules."""
    n = pos.shape[0]
    tree = cKDTree(pos)
    pairs = tree.query_pairs(rc, output_type="ndarray")
    a, b = pairs[:, 0], pairs[:, 1]
    if mol_ptr is not None:
        mol = np.searchsorted(mol_ptr, np.arange(n), side="right") - 1
        same = mol[a] == mol[b]
        a, b = a[same], b[same]
    d = pos[b] - pos[a]
    r = np.sqrt((d * d).sum(1))
    keep = (r > 0) & (r < rc)
    a, b, d = a[keep], b[keep], d[keep]
    return _csr_from_pairs(n, np.concatenate([a, b]), np.concatenate([b, a]), np.concatenate([d, -d]))


def molecules(seed, n_mol, size_lo=15, size_hi=80, bond_lo=1.0, bond_hi=1.5, min_dist=0.9):
    """Random bonded growth: atom 0 at the origin; then repeatedly a uniform random existing
    parent, an isotropic direction, a bond length U[bond_lo, bond_hi]; reject a candidate closer
    than min_dist to any atom of the molecule.  Molecules are laid out 100 A apart on a line so
    a global neighbour search can never connect them (edges are also filtered by mol_ptr)."""
    sizes = rng.randint(seed, rng.STREAMS["mol_size"], np.arange(n_mol), size_lo, size_hi)
    mol_ptr = np.zeros(n_mol + 1, dtype=np.int32)
    mol_ptr[1:] = np.cumsum(sizes)
    pos = np.zeros((int(mol_ptr[-1]), 3))
    for m in range(n_mol):
        base = mol_ptr[m]
        size = int(sizes[m])
        p = np.zeros((size, 3))
        cnt = 1
        k = np.uint64(m) << np.uint64(32)
        while cnt < size:
            parent = int(rng.uniform(seed, rng.STREAMS["mol_parent"], k) * cnt)
            dirn = rng.normal(seed, rng.STREAMS["mol_dir"], (3,), offset=int(3 * k))
            dirn = dirn / np.linalg.norm(dirn)
            bond = bond_lo + (bond_hi - bond_lo) * float(rng.uniform(seed, rng.STREAMS["mol_bond"], k))
            cand = p[parent] + bond * dirn
            k += np.uint64(1)
            d = p[:cnt] - cand
            if np.min((d * d).sum(1)) < min_dist * min_dist:
                continue
            p[cnt] = cand
            cnt += 1
        pos[base:base + size] = p + np.array([100.0 * m, 0.0, 0.0])
    return pos, mol_ptr
