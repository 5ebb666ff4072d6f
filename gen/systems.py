"""Seeded synthetic atom systems shaped like the paper's workloads (BASELINE.json `configs`).

Only geometry sampling lives here (uniform draws, rejection by distance, lattice construction, periodic
image bookkeeping).  No basis functions, cutoffs, filters or model arithmetic.

Species indices: configs 1-3 {O:0, H:1}; config 4 {X:0}; config 5 {H:0, C:1, N:2, O:3, S:4}.
All generators emit positions wrapped into [0, L) (ghost images lie outside by construction).
"""
from __future__ import annotations

import numpy as np
from scipy.spatial import cKDTree

OH_BOND = 0.96
HOH_ANGLE = np.deg2rad(104.5)

# model hyper-parameters and default sizes per BASELINE.json config (1-based index)
CONFIGS = {
    1: dict(name="tiny_water_192", n_species=2, F=32, K=16, T=2, rc=5.0, seed=101, wseed=1001,
            n_mol=64, L=12.42),
    # literal L=43.1 A is 3x water density and makes the O-O>=2.5 A rejection unsatisfiable
    # (SURVEY.md §8(d)); corrected box keeps 24,000 atoms at ~52 neighbours/atom.
    2: dict(name="bulk_water_24k", n_species=2, F=128, K=20, T=3, rc=5.0, seed=102, wseed=1002,
            n_mol=8000, L=62.08),
    3: dict(name="slab_96k", n_species=2, F=128, K=20, T=3, rc=5.0, seed=103, wseed=1002,
            n_mol=32000, L=98.55, halo=5.0),
    4: dict(name="diamond_512k", n_species=1, F=128, K=20, T=3, rc=5.0, seed=104, wseed=1004,
            ncell=40, a=5.43, sigma=0.05),
    5: dict(name="peptide_water_1M", n_species=5, F=128, K=20, T=3, rc=5.0, seed=105, wseed=1005,
            n_slots=343000, L=217.3, chain_frac=0.02, chain_len=20),
}


def _unit_vectors(rng, n):
    a = rng.standard_normal((n, 3))
    a /= np.linalg.norm(a, axis=1, keepdims=True)
    return a


def _rsa(rng, n_target, lo, hi, boxsize, dmin, exclude=None, dmin_excl=0.0):
    """Batched random sequential placement of n_target points uniform in [lo,hi) rejecting any pair closer
    than dmin (periodic with `boxsize`).  Conservative batch rule: a candidate is dropped when ANY
    lower-index candidate of the same batch is within dmin (accepted or not)."""
    lo = np.asarray(lo, float)
    hi = np.asarray(hi, float)
    acc = np.empty((0, 3))
    excl_tree = cKDTree(exclude, boxsize=boxsize) if exclude is not None and len(exclude) else None
    stall = 0
    while len(acc) < n_target:
        need = n_target - len(acc)
        m = int(min(max(8 * need, 4096), 2_000_000))
        cand = lo + (hi - lo) * rng.random((m, 3))
        if len(acc):
            dn, _ = cKDTree(acc, boxsize=boxsize).query(cand, k=1, distance_upper_bound=dmin, workers=-1)
            cand = cand[~np.isfinite(dn)]
        if excl_tree is not None and len(cand):
            dn, _ = excl_tree.query(cand, k=1, distance_upper_bound=dmin_excl, workers=-1)
            cand = cand[~np.isfinite(dn)]
        if len(cand) > 1:
            pairs = cKDTree(cand, boxsize=boxsize).query_pairs(dmin, output_type="ndarray")
            rej = np.zeros(len(cand), bool)
            if len(pairs):
                rej[np.maximum(pairs[:, 0], pairs[:, 1])] = True
            cand = cand[~rej]
        stall = stall + 1 if len(cand) == 0 else 0
        if stall > 200:
            raise RuntimeError("random sequential placement saturated; density too high for dmin")
        acc = np.concatenate([acc, cand[:need]])
    return acc


def _add_hydrogens(rng, O):
    n = len(O)
    a = _unit_vectors(rng, n)
    t = _unit_vectors(rng, n)
    b = t - (t * a).sum(1, keepdims=True) * a
    b /= np.linalg.norm(b, axis=1, keepdims=True)
    h1 = O + OH_BOND * a
    h2 = O + OH_BOND * (np.cos(HOH_ANGLE) * a + np.sin(HOH_ANGLE) * b)
    return np.stack([O, h1, h2], axis=1).reshape(3 * n, 3)


def water_box(n_mol, box, seed, zlo=None, zhi=None, type_O=0, type_H=1, exclude=None, dmin_excl=0.0,
              rng=None):
    """n_mol water-like molecules: O by random sequential placement rejecting O-O < 2.5 A (periodic),
    H at 0.96 A in uniformly random orientation with H-O-H = 104.5 deg.  Returns (pos[3n,3], types[3n])."""
    rng = np.random.Generator(np.random.PCG64(seed)) if rng is None else rng
    box = np.asarray(box, float)
    lo = np.zeros(3)
    hi = box.copy()
    if zlo is not None:
        lo[2], hi[2] = zlo, zhi
    O = _rsa(rng, n_mol, lo, hi, box, 2.5, exclude=exclude, dmin_excl=dmin_excl)
    pos = _add_hydrogens(rng, O)
    pos -= np.floor(pos / box) * box
    pos = np.where(pos >= box, 0.0, pos)          # guard x == L after rounding
    types = np.tile(np.array([type_O, type_H, type_H], np.int32), n_mol)
    return pos, types


def diamond(ncell, a, sigma, seed):
    """Diamond-cubic lattice, ncell^3 conventional cells (8 atoms each), Gaussian displacement sigma per
    component.  Returns (pos, types, box)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    basis = np.array([[0, 0, 0], [0, .5, .5], [.5, 0, .5], [.5, .5, 0],
                      [.25, .25, .25], [.25, .75, .75], [.75, .25, .75], [.75, .75, .25]])
    g = np.arange(ncell)
    cells = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 1, 3)
    pos = ((cells + basis[None]) * a).reshape(-1, 3)
    if sigma > 0:
        pos = pos + sigma * rng.standard_normal(pos.shape)
    box = np.full(3, ncell * a)
    pos -= np.floor(pos / box) * box
    pos = np.where(pos >= box, 0.0, pos)
    return pos, np.zeros(len(pos), np.int32), box


def periodic_ghosts(pos, box, halo, periodic=(True, True, True)):
    """All periodic images (S != 0) of the given atoms that lie within `halo` outside a face of the box,
    i.e. inside [-halo, L+halo)^3 but not the box itself.  Returns (ghost_pos, ghost_owner, ghost_image)."""
    box = np.asarray(box, float)
    smax = [int(np.ceil(halo / box[d])) if periodic[d] else 0 for d in range(3)]
    gp, go, gi = [], [], []
    idx = np.arange(len(pos))
    for sx in range(-smax[0], smax[0] + 1):
        for sy in range(-smax[1], smax[1] + 1):
            for sz in range(-smax[2], smax[2] + 1):
                if sx == 0 and sy == 0 and sz == 0:
                    continue
                S = np.array([sx, sy, sz])
                p = pos + S * box
                m = np.all((p >= -halo) & (p < box + halo), axis=1)
                if m.any():
                    gp.append(p[m]); go.append(idx[m]); gi.append(np.broadcast_to(S, (m.sum(), 3)))
    if not gp:
        return np.empty((0, 3)), np.empty(0, np.int32), np.empty((0, 3), np.int8)
    return np.concatenate(gp), np.concatenate(go).astype(np.int32), np.concatenate(gi).astype(np.int8)


def slab_with_ghosts(n_mol, L, halo, seed):
    """Liquid-vapour slab: water in z in [0, L] of an L x L x 3L periodic box, empty above; ghosts = periodic
    images within `halo` outside the faces, with owner map (open-boundary / ghost mode)."""
    box = np.array([L, L, 3 * L])
    pos, types = water_box(n_mol, box, seed, zlo=1.0, zhi=L - 1.0)
    gpos, gown, _ = periodic_ghosts(pos, box, halo)
    allpos = np.concatenate([pos, gpos])
    alltypes = np.concatenate([types, types[gown]]).astype(np.int32)
    return allpos, alltypes, box, len(pos), len(gpos), gown


class _HashGrid:
    def __init__(self, box, h):
        self.box = box
        self.n = np.maximum((box / h).astype(int), 1)
        self.h = box / self.n
        self.cells = {}

    def _key(self, p):
        c = np.floor(p / self.h).astype(int) % self.n
        return int(c[0]), int(c[1]), int(c[2])

    def add(self, p):
        self.cells.setdefault(self._key(p), []).append(p)

    def clash(self, p, dmin):
        c = np.floor(p / self.h).astype(int)
        d2 = dmin * dmin
        for dx in (-1, 0, 1):
            for dy in (-1, 0, 1):
                for dz in (-1, 0, 1):
                    k = ((c[0] + dx) % self.n[0], (c[1] + dy) % self.n[1], (c[2] + dz) % self.n[2])
                    for q in self.cells.get(k, ()):
                        d = p - q
                        d -= self.box * np.round(d / self.box)
                        if d @ d < d2:
                            return True
        return False


def peptide_water(n_slots, L, chain_frac, chain_len, seed):
    """~1M-atom solvated-peptide-like mixture: chain_frac of the molecule slots are replaced by chains of
    chain_len atoms (species uniform over {H,C,N,O,S}, 1.5 A random-walk bonds, no atom closer than 1.2 A to
    any other); the rest is water (O=3, H=0) placed as in water_box, O kept >= 2.16 A from chain atoms so no
    water atom comes within 1.2 A of a chain atom."""
    rng = np.random.Generator(np.random.PCG64(seed))
    box = np.full(3, float(L))
    n_rep = int(round(chain_frac * n_slots))
    n_chain = (3 * n_rep) // chain_len
    n_rep = (n_chain * chain_len) // 3
    assert n_chain * chain_len == 3 * n_rep, "chain atoms must fill whole molecule slots"
    grid = _HashGrid(box, 1.5)
    cpos = []
    for _ in range(n_chain):
        while True:
            chain = []
            p = rng.random(3) * box
            ok = not grid.clash(p, 1.2)
            if ok:
                chain.append(p)
                while len(chain) < chain_len:
                    for _try in range(64):
                        q = chain[-1] + 1.5 * _unit_vectors(rng, 1)[0]
                        q -= np.floor(q / box) * box
                        if grid.clash(q, 1.2):
                            continue
                        if any(((lambda d: d @ d)((q - r) - box * np.round((q - r) / box)) < 1.44)
                               for r in chain):
                            continue
                        chain.append(q)
                        break
                    else:
                        ok = False
                        break
            if ok:
                break
        for p in chain:
            grid.add(p)
        cpos.extend(chain)
    cpos = np.array(cpos).reshape(-1, 3)
    ctypes_ = rng.integers(0, 5, size=len(cpos)).astype(np.int32)
    wpos, wtypes = water_box(n_slots - n_rep, box, seed=None, type_O=3, type_H=0,
                             exclude=cpos, dmin_excl=1.2 + OH_BOND, rng=rng)
    pos = np.concatenate([cpos, wpos])
    pos = np.where(pos >= box, 0.0, pos)
    return pos, np.concatenate([ctypes_, wtypes]).astype(np.int32), box


def replicate(pos, types, box, reps=(2, 2, 2)):
    """Periodic replication (used by the extensivity pin)."""
    box = np.asarray(box, float)
    out_p, out_t = [], []
    for ix in range(reps[0]):
        for iy in range(reps[1]):
            for iz in range(reps[2]):
                out_p.append(pos + np.array([ix, iy, iz]) * box)
                out_t.append(types)
    return np.concatenate(out_p), np.concatenate(out_t), box * np.array(reps)


def extract_cluster(pos, box, center, r_local, r_total):
    """Atoms within r_total of atom `center` (minimum image if box is given), unwrapped around the centre.
    Returns (idx_local, idx_ghost, cluster_pos) with locals (dist < r_local) first.  Needs r_total < L/2."""
    d = pos - pos[center]
    if box is not None:
        box = np.asarray(box, float)
        assert r_total < box.min() / 2
        d = d - box * np.round(d / box)
    dist = np.linalg.norm(d, axis=1)
    il = np.nonzero(dist < r_local)[0]
    ig = np.nonzero((dist >= r_local) & (dist < r_total))[0]
    idx = np.concatenate([il, ig])
    return il, ig, pos[center] + d[idx]


def random_gas(n, box, dmin, seed, n_species=2, empty_frac=0.0):
    """n uniform points in an orthorhombic periodic box with no pair closer than dmin (draw, drop the later atom of every
    close pair, redraw the missing ones); `empty_frac` keeps the top of the box in z empty.  Row-length stress input
    for the neighbour list and the edge kernels: far from the paper's liquids on both sides (isolated atoms at low
    density, rows of > 100 neighbours at high density)."""
    rng = np.random.default_rng(seed)
    box = np.asarray(box, float)
    hi = box * np.array([1.0, 1.0, 1.0 - empty_frac])
    pos = np.empty((0, 3))
    for _ in range(200):
        pos = np.vstack([pos, rng.uniform(0.0, 1.0, (n - len(pos), 3)) * hi])
        pairs = cKDTree(pos, boxsize=box).query_pairs(dmin, output_type="ndarray")
        if len(pairs) == 0:
            break
        keep = np.ones(len(pos), bool)
        keep[pairs[:, 1]] = False                      # i < j in every pair: the earlier atom stays
        pos = pos[keep]
    assert len(pos) == n, "random_gas: density too high for dmin"
    types = rng.integers(0, n_species, n).astype(np.int32)
    return np.ascontiguousarray(pos), types, box


def make_config(k, **over):
    """Build BASELINE.json config k (1..5).  Size overrides (n_mol, L, ncell, n_slots, ...) give the reduced
    variants the CPU tests use.  Returns a dict: pos, types, box, n_local, n_ghost, ghost_owner, model."""
    c = dict(CONFIGS[k]); c.update(over)
    model = dict(n_species=c["n_species"], F=c["F"], K=c["K"], T=c["T"], rc=c["rc"], wseed=c["wseed"])
    ghost_owner = None
    if k in (1, 2):
        box = np.full(3, float(c["L"]))
        pos, types = water_box(c["n_mol"], box, c["seed"])
        n_local, n_ghost = len(pos), 0
    elif k == 3:
        pos, types, box, n_local, n_ghost, ghost_owner = slab_with_ghosts(c["n_mol"], c["L"], c["halo"], c["seed"])
    elif k == 4:
        pos, types, box = diamond(c["ncell"], c["a"], c["sigma"], c["seed"])
        n_local, n_ghost = len(pos), 0
    elif k == 5:
        pos, types, box = peptide_water(c["n_slots"], c["L"], c["chain_frac"], c["chain_len"], c["seed"])
        n_local, n_ghost = len(pos), 0
    else:
        raise KeyError(k)
    return dict(name=c["name"], pos=np.ascontiguousarray(pos), types=np.ascontiguousarray(types, np.int32),
                box=np.asarray(box, float), n_local=int(n_local), n_ghost=int(n_ghost),
                ghost_owner=ghost_owner, model=model)
