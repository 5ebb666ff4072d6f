"""Neighbour-list management of the deployed path:

  * Verlet skin: the list is built at rc + skin, every step re-filters it at rc ("drop edges longer than the cutoff each
    step") and a full rebuild happens only when an atom has moved further than skin / 2; steps that reuse the list are
    replayed from a captured CUDA graph.  Along a trajectory the edge SET of every step must be bit-identical to the
    oracle's brute-force set, and E / F / W must match the oracle and the rebuild-every-step path.
  * T-hop pruning in ghost mode: atoms no local atom reaches within T hops are dropped and layer t only updates the atoms
    within T - 1 - t hops; "pruning does not change the result, only the cost".
  * Re-entrancy: options belong to the model; two models with different options on two host threads.
"""
import threading

import numpy as np
import pytest

import gen
import oracle
from test_gpu_parity import SMALL, _blob, _check, _oracle_eval, _same_edges, _torch

pytestmark = pytest.mark.gpu


def _sorted_edges(i, j, im):
    order = np.lexsort((im[:, 2], im[:, 1], im[:, 0], j, i))
    return i[order], j[order], im[order]


def _run(m, pos, types, box, n_local=None, n_ghost=0, owner=None):
    torch = _torch()
    dev = torch.device("cuda:0")
    e, f, w = m.compute(torch.from_numpy(np.ascontiguousarray(pos)).to(dev), torch.from_numpy(types).to(dev), box, n_local, n_ghost,
                        None if owner is None else torch.from_numpy(np.ascontiguousarray(owner, np.int32)).to(dev))
    torch.cuda.synchronize()
    return float(e[0]), f.cpu().numpy(), w.cpu().numpy()


@pytest.mark.parametrize("k,skin_mA,step_A", [(1, 2000, 0.04), (2, 1000, 0.04), (5, 500, 0.015)])
def test_skin_reuse_trajectory_matches_rebuild_and_oracle(k, skin_mA, step_A):
    """20 steps of a random walk (step_A per step and component, atoms wrapped back into the box when they leave it).  The
    skin list must be reused on most steps and rebuilt when the displacement criterion says so; every step: edge set ==
    oracle set (bit-exact), E / F / W within tolerance of the oracle, and equal (to fp32 summation order) to a model that
    rebuilds every step."""
    import paper_2506_04055_b200 as P
    c = gen.make_config(k, **SMALL[k])
    blob = _blob(c["model"])
    mdl = c["model"]
    N = len(c["pos"])
    box = np.asarray(c["box"], np.float64)
    rng = np.random.default_rng(100 + k)
    pos = c["pos"].copy()
    with P.Model(blob, mdl["n_species"], mdl["rc"], N) as ms, P.Model(blob, mdl["n_species"], mdl["rc"], N) as m0:
        ms.set_option("skin_mA", skin_mA)
        m0.set_option("skin_mA", 0)
        for step in range(20):
            es, fs, ws = _run(ms, pos, c["types"], box)
            e0, f0, w0 = _run(m0, pos, c["types"], box)
            gi, gj, gim = ms.neighbors()
            hi, hj, him = m0.neighbors()
            assert np.array_equal(gi, hi) and np.array_equal(gj, hj) and np.array_equal(gim, him), step
            # the two paths differ in the row order (= fp32 summation order) only: forces agree far inside the tolerance;
            # each is held to the oracle (the energy of these random-weight models amplifies rounding, B1)
            frms = np.sqrt((f0 ** 2).mean())
            assert np.abs(fs - f0).max() <= 5e-3 * frms, (step, np.abs(fs - f0).max() / frms)
            if step % 3 == 0 or step == 19:
                oi, oj, oim = oracle.neighbors(pos, box, mdl["rc"])
                assert np.array_equal(gi, oi) and np.array_equal(gj, oj) and np.array_equal(gim, oim), step
                ref = oracle.compute(blob, pos, c["types"], box)
                _check(c, es, fs, ws, ref, f"config {k} skin {skin_mA} mA step {step}")
                _check(c, e0, f0, w0, ref, f"config {k} rebuild every step, step {step}")
            pos = pos + step_A * rng.standard_normal(pos.shape)
            pos -= np.floor(pos / box) * box                    # the caller re-wraps: as-given coordinates jump by a box length
        st = ms.stats()
        print(f"config {k}: rebuilds {st['n_list_rebuilds']} reuses {st['n_list_reuses']} graph replays {st['n_graph_replays']}")
        assert st["n_list_rebuilds"] + st["n_list_reuses"] == 20
        assert st["n_list_reuses"] >= 10 and st["n_list_rebuilds"] >= 1
        assert st["n_graph_replays"] >= 5
        assert m0.stats()["n_list_rebuilds"] == 20 and m0.stats()["n_list_reuses"] == 0


def test_skin_static_positions_replay_is_bit_identical():
    import paper_2506_04055_b200 as P
    c = gen.make_config(2, **SMALL[2])
    blob = _blob(c["model"])
    mdl = c["model"]
    with P.Model(blob, mdl["n_species"], mdl["rc"], len(c["pos"])) as m:
        m.set_option("skin_mA", 1500)
        out = [_run(m, c["pos"], c["types"], c["box"]) for _ in range(4)]
        st = m.stats()
    assert st["n_list_rebuilds"] == 1 and st["n_list_reuses"] == 3 and st["n_graph_replays"] == 3
    for e, f, w in out[1:]:
        assert e == out[0][0] and np.array_equal(w, out[0][2]) and np.abs(f - out[0][1]).max() <= 1e-9 * np.abs(f).max()


def test_skin_with_ghosts_and_owner_fold():
    """Open-boundary list (no wrap bookkeeping) with the fold; ghosts move with their owners."""
    import paper_2506_04055_b200 as P
    c = gen.make_config(3, **SMALL[3])
    blob = _blob(c["model"])
    mdl = c["model"]
    N, nl = len(c["pos"]), c["n_local"]
    rng = np.random.default_rng(7)
    pos = c["pos"].copy()
    own = np.asarray(c["ghost_owner"], np.int64)
    with P.Model(blob, mdl["n_species"], mdl["rc"], N) as m:
        m.set_option("skin_mA", 1000)
        for step in range(6):
            e, f, w = _run(m, pos, c["types"], c["box"], nl, c["n_ghost"], c["ghost_owner"])
            if step in (0, 3, 5):
                ref = oracle.compute(blob, pos, c["types"], c["box"], nl, c["n_ghost"], c["ghost_owner"])
                cc = dict(c); cc["pos"] = pos
                _same_edges(m, cc)                       # the pruned sub-graph of the oracle's set, bit-exact
                _check(c, e, f, w, ref, f"slab + ghosts, skin, step {step}")
            d = 0.03 * rng.standard_normal((nl, 3))
            pos[:nl] += d
            pos[nl:] += d[own]
        st = m.stats()
        assert st["n_list_reuses"] >= 4


@pytest.mark.parametrize("halo,fold", [(5.0, True), (5.0, False), (15.0, True)])
def test_thop_pruning_does_not_change_the_result(halo, fold):
    """Ghost mode with a 1 rc halo (config 3's recipe: a truncated graph) and with the complete T rc = 15 A halo: pruned ==
    un-pruned == oracle (E, folded or partial F, W), fewer atoms kept, and the stray images nobody reaches get zero force."""
    import paper_2506_04055_b200 as P
    c = gen.make_config(3, n_mol=600, L=26.2, halo=halo)
    blob = _blob(c["model"])
    mdl = c["model"]
    N, nl = len(c["pos"]), c["n_local"]
    own = c["ghost_owner"] if fold else None
    ref = oracle.compute(blob, c["pos"], c["types"], c["box"], nl, c["n_ghost"], own)
    res = {}
    for prune in (1, 0):
        with P.Model(blob, mdl["n_species"], mdl["rc"], N) as m:
            m.set_option("prune", prune)
            m.set_option("skin_mA", 0)
            e, f, w = _run(m, c["pos"], c["types"], c["box"], nl, c["n_ghost"], own)
            st = m.stats()
            res[prune] = (e, f, w, st)
        _check(c, e, f, w, ref, f"slab halo {halo} fold {fold} prune {prune} (kept {st['n_reached']} of {N})")
    e1, f1, w1, st1 = res[1]
    e0, f0, w0, st0 = res[0]
    assert st0["n_reached"] == N and st1["n_reached"] <= N
    frms = np.sqrt((f0 ** 2).mean())
    assert abs(e1 - e0) <= 2e-4 * nl and np.abs(f1 - f0).max() <= 1e-2 * frms and np.allclose(w1, w0, rtol=2e-3, atol=2e-3 * np.abs(w0).max())
    if halo > 10.0:
        assert st1["n_reached"] < N          # images of the bottom layer at the top of the empty box reach nobody
    # the pruned list is the sub-graph over the reached atoms; un-pruned it is the oracle's full set
    assert st0["n_edges"] == ref["n_edges"] and st1["n_edges"] <= st0["n_edges"]
    oi, oj, _ = oracle.neighbors(c["pos"], c["box"], mdl["rc"], periodic=False)
    from test_gpu_parity import reached_atoms
    keep = reached_atoms(oi, oj, nl, N, mdl["T"])
    assert st1["n_reached"] == int(keep.sum()) and st1["n_edges"] == int((keep[oi] & keep[oj]).sum())
    if not fold:
        assert not f1[~keep].any()             # dropped atoms get exactly zero partial force


def test_pruning_and_skin_together():
    import paper_2506_04055_b200 as P
    c = gen.make_config(3, n_mol=600, L=26.2, halo=15.0)
    blob = _blob(c["model"])
    mdl = c["model"]
    N, nl = len(c["pos"]), c["n_local"]
    rng = np.random.default_rng(11)
    pos = c["pos"].copy()
    own = np.asarray(c["ghost_owner"], np.int64)
    with P.Model(blob, mdl["n_species"], mdl["rc"], N) as m:
        m.set_option("skin_mA", 1000)
        for step in range(5):
            e, f, w = _run(m, pos, c["types"], c["box"], nl, c["n_ghost"], c["ghost_owner"])
            if step in (0, 4):
                ref = oracle.compute(blob, pos, c["types"], c["box"], nl, c["n_ghost"], c["ghost_owner"])
                _check(c, e, f, w, ref, f"15 A halo, pruned + skin, step {step}")
            d = 0.03 * rng.standard_normal((nl, 3))
            pos[:nl] += d
            pos[nl:] += d[own]
        st = m.stats()
        assert st["n_list_reuses"] >= 3 and st["n_reached"] < N


def test_two_models_two_threads_different_options():
    """Options live in the model (no process-wide state): two models with different implementation switches evaluate
    concurrently from two host threads, each on its own stream, and both match the oracle."""
    import paper_2506_04055_b200 as P
    torch = _torch()
    dev = torch.device("cuda:0")
    c = gen.make_config(5, **SMALL[5])
    blob = _blob(c["model"])
    mdl = c["model"]
    ref = _oracle_eval(c, blob)
    pos = torch.from_numpy(c["pos"]).to(dev)
    types = torch.from_numpy(c["types"]).to(dev)
    opts = [dict(), dict(edge_path=1, gemm_fwd_exact=0, atoms_per_unit=7, skin_mA=0)]
    out = [None, None]
    err = []

    def work(k):
        try:
            st = torch.cuda.Stream(device=dev)
            with P.Model(blob, mdl["n_species"], mdl["rc"], len(c["pos"])) as m:
                for name, v in opts[k].items():
                    m.set_option(name, v)
                for _ in range(6):
                    with torch.cuda.stream(st):
                        e, f, w = m.compute(pos, types, c["box"], stream=st)
                    st.synchronize()
                out[k] = (float(e[0]), f.cpu().numpy(), w.cpu().numpy())
        except Exception as ex:                      # noqa: BLE001
            err.append(ex)

    th = [threading.Thread(target=work, args=(k,)) for k in range(2)]
    for t in th:
        t.start()
    for t in th:
        t.join()
    assert not err, err
    for k in range(2):
        _check(c, *out[k], ref, f"thread {k} options {opts[k]}")
    assert out[0][0] != out[1][0]                    # different kernels did run (plain fp32 edge path vs tensor-core path)


def test_list_is_rebuilt_when_the_system_changes():
    """The kept list serves a call only for the same atom counts, species and box, and only while no atom has moved further
    than skin / 2: each of these changes must rebuild (and give the oracle's result)."""
    import paper_2506_04055_b200 as P
    c = gen.make_config(1)
    blob = _blob(c["model"])
    mdl = c["model"]
    N = len(c["pos"])
    with P.Model(blob, mdl["n_species"], mdl["rc"], N) as m:
        m.set_option("skin_mA", 1500)
        _run(m, c["pos"], c["types"], c["box"])
        _run(m, c["pos"], c["types"], c["box"])
        assert (m.stats()["n_list_rebuilds"], m.stats()["n_list_reuses"]) == (1, 1)
        # (i) one atom jumps by 1 A > skin / 2
        pos = c["pos"].copy(); pos[17, 1] += 1.0
        e, f, w = _run(m, pos, c["types"], c["box"])
        assert m.stats()["n_list_rebuilds"] == 2
        _check(c, e, f, w, oracle.compute(blob, pos, c["types"], c["box"]), "jump > skin / 2")
        # (ii) a species changes
        types = c["types"].copy(); types[5] = 1 - types[5]
        e, f, w = _run(m, pos, types, c["box"])
        assert m.stats()["n_list_rebuilds"] == 3
        _check(c, e, f, w, oracle.compute(blob, pos, types, c["box"]), "species change")
        # (iii) the box changes (positions scaled with it)
        box2 = np.asarray(c["box"]) * 1.01
        e, f, w = _run(m, pos * 1.01, types, box2)
        assert m.stats()["n_list_rebuilds"] == 4
        _check(c, e, f, w, oracle.compute(blob, pos * 1.01, types, box2), "box change")
        # (iv) fewer atoms
        e, f, w = _run(m, pos[:150] * 1.01, types[:150], box2)
        assert m.stats()["n_list_rebuilds"] == 5 and f.shape == (150, 3)
        cc = dict(c); cc["n_local"] = 150
        _check(cc, e, f, w, oracle.compute(blob, pos[:150] * 1.01, types[:150], box2), "fewer atoms")
        # ... and then it is reused again
        _run(m, pos[:150] * 1.01, types[:150], box2)
        assert m.stats()["n_list_reuses"] == 2


def test_host_entry_point_with_list_reuse():
    import paper_2506_04055_b200 as P
    c = gen.make_config(2, **SMALL[2])
    blob = _blob(c["model"])
    mdl = c["model"]
    with P.Model(blob, mdl["n_species"], mdl["rc"], len(c["pos"])) as m:
        out = [m.compute_host(c["pos"], c["types"], c["box"]) for _ in range(3)]
        out = [(float(e[0]), f.copy(), w.copy()) for e, f, w in out]
        st = m.stats()
    assert st["n_list_rebuilds"] == 1 and st["n_list_reuses"] == 2 and st["n_graph_replays"] == 2
    assert out[1][0] == out[0][0] == out[2][0] and np.abs(out[2][1] - out[0][1]).max() <= 1e-9 * np.abs(out[0][1]).max()
    _check(c, *out[2], _oracle_eval(c, blob), "host entry point, third call (graph replay)")


@pytest.mark.parametrize("k", [1, 2])
def test_rigid_drift_far_out_of_the_box(k):
    """The MD protocol leg of bench.py: the whole configuration drifts rigidly by 0.048 A per step and is never
    wrapped by the caller -- after 150 steps every atom has left the box by up to 7.2 A (config 1: more than half a box length).
    Pair vectors do not change, so at EVERY step the (i, j, image) set is the one of step 0 (images are relative to the positions
    as given), E / F / W stay at their step-0 values up to the fp32 rounding of the shifted coordinates, and the kept list is
    rebuilt exactly when the displacement since the last build exceeds skin / 2 (every 11 steps at skin 1 A), replaying the
    captured graph in between."""
    import paper_2506_04055_b200 as P
    c = gen.make_config(k, **SMALL[k])
    blob = _blob(c["model"])
    mdl = c["model"]
    N = len(c["pos"])
    box = np.asarray(c["box"], np.float64)
    v = 0.048 * np.array([0.6, 0.64, 0.48])                  # |v| = 0.048 A per step
    pos = c["pos"].copy()
    with P.Model(blob, mdl["n_species"], mdl["rc"], N) as m:
        m.set_option("skin_mA", 1000)
        e0, f0, w0 = _run(m, pos, c["types"], box)
        ref_edges = m.neighbors()
        frms = np.sqrt((f0 ** 2).mean())
        for step in range(1, 151):
            pos += v
            e, f, w = _run(m, pos, c["types"], box)
            assert abs(e - e0) <= 1e-4 * N, (step, e, e0)
            assert np.sqrt(((f - f0) ** 2).mean()) <= 2e-4 * frms and np.abs(f - f0).max() <= 2e-3 * frms, step
            assert np.linalg.norm(w - w0) <= 2e-4 * np.linalg.norm(w0), step
            if step % 7 == 0 or step > 140:
                for x, y in zip(m.neighbors(), ref_edges):
                    assert np.array_equal(x, y), step
        st = m.stats()
    # displacement after n steps = 0.048 n: 0.48 A at n = 10, 0.528 > skin / 2 at n = 11, i.e. a rebuild at steps 11, 22, ... (+ the build at step 0)
    assert st["n_list_rebuilds"] == 1 + 150 // 11, st
    assert st["n_list_reuses"] == 150 - 150 // 11 and st["n_graph_replays"] >= st["n_list_reuses"] - 2, st
