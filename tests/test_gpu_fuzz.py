"""Randomised parity: small random systems (1 .. 1,500 atoms, three densities, 1-6 species), random model shapes
(F in {32, 64, 128}, K in {8, 16, 20, 23}, T <= 3: every kernel family incl. the species-table fallbacks of the layer-0
passes), periodic or ghost mode (halo 5 / 7.5 / 15 A, with and without owner fold), random skin / pruning options, atom
capacity too small on purpose (regrow), short random-walk trajectories with re-wrapped coordinates -- every step against the
fp64 oracle: edge set, E, F, W.  Fixed seeds, 100 cases each (about 20 s).  (Developed as a long-running fuzz: ~3,600 cases over five
seeds without a logic failure; 4-layer F = 128 models on dense random gases were excluded -- they are ill-conditioned in
fp32 on EVERY kernel path, plain FFMA included.)"""
import numpy as np
import pytest

import gen
import oracle
from test_gpu_parity import _torch, reached_atoms

pytestmark = pytest.mark.gpu


def _edge_set(i, j, im):
    return set(zip(i.tolist(), j.tolist(), map(tuple, im.tolist())))


@pytest.mark.parametrize("seed", [11, 12])
def test_random_systems_options_and_trajectories(seed):
    import paper_2506_04055_b200 as P
    torch = _torch()
    dev = torch.device("cuda:0")
    rng = np.random.default_rng(seed)
    n_case = n_ghost_cases = 0
    while n_case < 100:                       # a fixed number of cases: the sequence is deterministic for a seed
        F = int(rng.choice([32, 64, 128, 128, 128])); K = int(rng.choice([8, 16, 20, 23])); T = int(rng.integers(1, 4))
        ns = int(rng.integers(1, 7))
        blob = gen.make_weights(ns, F, K, T, 5.0, seed=int(rng.integers(1 << 30)))
        n = int(rng.choice([1, 2, 7, 33, 200, 700, 1500]))
        dens = float(rng.choice([0.005, 0.03, 0.1]))
        L = max((n / dens) ** (1 / 3), 10.5)
        box = np.array([L, L * float(rng.uniform(1, 1.4)), L * float(rng.uniform(1, 1.8))])
        try:
            pos, types, box = gen.random_gas(n, box, 1.1, seed=int(rng.integers(1 << 30)), n_species=ns)
        except AssertionError:
            continue
        ghost = rng.random() < 0.4 and n >= 33
        skin = int(rng.choice([0, 300, 1000, 2500])); prune = int(rng.integers(0, 2))
        go = owner = None
        apos, atypes, nl, ng = pos, types, n, 0
        if ghost:
            gp, go, _ = gen.periodic_ghosts(pos, box, float(rng.choice([5.0, 7.5, 15.0])))
            if len(gp) == 0:
                continue
            apos = np.concatenate([pos, gp]); atypes = np.concatenate([types, types[go]]).astype(np.int32)
            ng = len(gp)
            owner = go.astype(np.int32) if rng.random() < 0.5 else None
            n_ghost_cases += 1
        n_case += 1
        label = f"seed {seed} case {n_case}: F{F} K{K} T{T} ns{ns} n{n}+{ng} dens{dens} skin{skin} prune{prune} fold{owner is not None}"
        with P.Model(blob, ns, 5.0, max(len(apos) // 2, 1)) as m:
            m.set_option("skin_mA", skin); m.set_option("prune", prune)
            p = apos.copy()
            for step in range(int(rng.integers(1, 5))):
                e, f, w = m.compute(torch.from_numpy(p).to(dev), torch.from_numpy(atypes).to(dev), box, nl, ng,
                                    None if owner is None else torch.from_numpy(owner).to(dev))
                torch.cuda.synchronize()
                e, f, w = float(e[0]), f.cpu().numpy(), w.cpu().numpy()
                ref = oracle.compute(blob, p, atypes, box, nl, ng, owner)
                gi, gj, gim = m.neighbors()
                oi, oj, oim = oracle.neighbors(p, box, 5.0, periodic=ng == 0)
                if ng > 0 and prune:
                    # kept graph = sub-graph over the atoms reached within T hops; with a skin the hop levels come from the
                    # rc + skin graph of the build (lower bounds), so a few more atoms may be kept
                    keep = reached_atoms(oi, oj, nl, len(p), T)
                    sel = keep[oi] & keep[oj]
                    G, O, Omin = _edge_set(gi, gj, gim), _edge_set(oi, oj, oim), _edge_set(oi[sel], oj[sel], oim[sel])
                    assert Omin <= G <= O and (skin > 0 or G == Omin), (label, step)
                else:
                    assert np.array_equal(gi, oi) and np.array_equal(gj, oj) and np.array_equal(gim, oim), (label, step)
                fr = ref["forces"]
                rms = np.sqrt((fr ** 2).mean()) if fr.size else 0.0
                de = abs(e - ref["energy"]) / max(nl, 1)
                # A17b / A17c: absolute 1e-4, the fp32-geometry floor of small replicas, 3e-5 relative for exploding models
                etol = max(1e-4, 3 * rms * 1.5e-7 / np.sqrt(max(nl, 1)), 3e-5 * abs(ref["energy"]) / max(nl, 1))
                assert np.isfinite(e) and np.isfinite(f).all() and np.isfinite(w).all(), (label, step)
                assert de <= etol, (label, step, de, etol)
                if rms > 0:
                    # A17d: absolute floor 1e-8 |E| per Angstrom -- a force that cancels to 1e-6 of its natural scale |E| / rc (one
                    # pair near the cutoff, caught where dE/dd changes sign: extended fuzz, seed 37) has no relative accuracy in fp32
                    ffloor = 1e-8 * abs(ref["energy"])
                    assert np.sqrt(((f - fr) ** 2).mean()) <= max(2e-3 * rms, ffloor), (label, step)
                    assert np.abs(f - fr).max() <= max(1e-2 * rms, 1e-3 * np.abs(fr).max(), 3 * ffloor), (label, step)
                wn = np.linalg.norm(ref["virial"])
                if wn > 0:
                    assert np.linalg.norm(w - ref["virial"]) <= 2e-3 * wn, (label, step)
                d = float(rng.choice([0.01, 0.03, 0.1])) * rng.standard_normal((nl, 3))
                p[:nl] += d
                if ng:
                    p[nl:] += d[go]
                elif rng.random() < 0.5:
                    p -= np.floor(p / box) * box
    print(f"seed {seed}: {n_case} cases ({n_ghost_cases} in ghost mode)")
    assert n_case == 100 and n_ghost_cases >= 10
