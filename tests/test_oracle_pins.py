"""Pins for the fp64 oracle (oracle/painn_oracle.c) against things OTHER than itself.

Each test targets a class of plausible mistakes (SURVEY.md §8(c) "What pins the oracle"):
  * finite differences of E            -> adjoint is the gradient of the forward (BASELINE.json north_star)
  * dense torch-autograd restatement   -> forward AND adjoint by an independent route (library autograd)
  * invariances    -> translation / rotation / reflection / permutation
  * Newton's third law, virial symmetry and W = -dE/d(strain)
  * extensivity under 2x2x2 replication (BASELINE.json)
  * ghost images with halo >= T*rc + owner fold == periodic result
  * closed forms: no-message model, dimer, continuity at the cutoff
  * neighbour set vs scipy cKDTree (library routine), symmetry, perfect diamond = 28 neighbours
"""
import numpy as np
import pytest

import gen
import oracle


def _blob(model, **kw):
    return gen.make_weights(model["n_species"], model["F"], model["K"], model["T"], model["rc"],
                            seed=model["wseed"], **kw)


def _small_water(n_mol=20, L=10.6, seed=7):
    box = np.full(3, L)
    pos, types = gen.water_box(n_mol, box, seed)
    return pos, types, box


SMALL_MODEL = dict(n_species=2, F=8, K=6, T=2, rc=5.0, wseed=11)


# ------------------------------------------------------------------ finite differences
def _fd_rows(args):
    """Worker of the finite-difference pin: 4th-order central differences of the oracle energy for a range of atoms.
    Runs in its own process with one OpenMP thread (a 192-atom evaluation does not scale over threads; eight
    single-threaded workers are ~3x faster than eight OpenMP threads on one evaluation at a time)."""
    blob, pos, types, box, lo, hi, h = args
    import oracle as orc
    out = np.zeros((hi - lo, 3))
    for a in range(lo, hi):
        for d in range(3):
            e = []
            for k in (1, -1, 2, -2):
                p = pos.copy(); p[a, d] += k * h
                e.append(orc.compute(blob, p, types, box)["energy"])
            out[a - lo, d] = -(8 * (e[0] - e[1]) - (e[2] - e[3])) / (12 * h)
    return lo, out


def _fd_init():
    import os
    os.environ["OMP_NUM_THREADS"] = "1"


def test_forces_match_finite_differences_config1(cfg1):
    """All 576 coordinates of config 1, |dF| <= 1e-6 (BASELINE.json).  4th-order central stencil at
    h = 1e-4 A (reading A21: the K = 16 basis makes the 2-point truncation term ~1e-6 itself)."""
    import multiprocessing as mp
    import os
    from concurrent.futures import ProcessPoolExecutor
    c = cfg1
    ref = oracle.compute(c["blob"], c["pos"], c["types"], c["box"])
    h = 1e-4
    n = c["pos"].shape[0]
    nw = max(1, min(os.cpu_count() or 1, 16))
    bounds = np.linspace(0, n, 4 * nw + 1).astype(int)
    jobs = [(c["blob"], c["pos"], c["types"], c["box"], int(bounds[i]), int(bounds[i + 1]), h)
            for i in range(len(bounds) - 1) if bounds[i + 1] > bounds[i]]
    F_fd = np.zeros_like(ref["forces"])
    with ProcessPoolExecutor(max_workers=nw, mp_context=mp.get_context("spawn"), initializer=_fd_init) as ex:
        for lo, out in ex.map(_fd_rows, jobs):
            F_fd[lo:lo + len(out)] = out
    err = np.abs(F_fd - ref["forces"]).max()
    assert err <= 1e-6, err


# ------------------------------------------------------------------ dense autograd restatement
def _dense_energy_torch(arrs, hdr, pos, types, box, n_local, periodic, states=None):
    """Independent restatement of SURVEY.md §8(c) Forward with dense masked pair tensors (no edge lists,
    no hand adjoint).  pos: torch fp64 [N,3] requiring grad; box torch [3].  `states` (a list) receives the layer
    states (s [N,F], v [N,3,F]) after the embedding and after every layer."""
    import torch
    F, K, T, rc, eps = hdr["F"], hdr["K"], hdr["T"], hdr["rc"], hdr["eps"]
    N = pos.shape[0]
    W = {k: torch.tensor(v, dtype=torch.float64) for k, v in arrs.items()}
    if periodic:
        g = torch.tensor([-1, 0, 1], dtype=torch.float64)
        S = torch.stack(torch.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3)      # [27,3]
    else:
        S = torch.zeros(1, 3, dtype=torch.float64)
    nS = S.shape[0]
    # r[i, j, S] = pos[j] + S*L - pos[i]
    r = pos[None, :, None, :] + (S * box)[None, None, :, :] - pos[:, None, None, :]        # [N,N,nS,3]
    d2 = (r * r).sum(-1)
    self_mask = torch.eye(N, dtype=torch.bool)[:, :, None] & (S.abs().sum(-1) == 0)[None, None, :]
    mask = (d2 < rc * rc) & ~self_mask                                                      # [N,N,nS]
    d = torch.sqrt(torch.where(mask, d2, torch.ones_like(d2)))
    u = r / d[..., None]
    n = torch.arange(1, K + 1, dtype=torch.float64)
    rho = torch.sin(n * torch.pi * d[..., None] / rc) / d[..., None]                       # [N,N,nS,K]
    fc = 0.5 * (1 + torch.cos(torch.pi * d / rc)) * mask                                   # masked cutoff
    silu = torch.nn.functional.silu
    s = W["Emb"][torch.as_tensor(types, dtype=torch.long)]                                  # [N,F]
    v = torch.zeros(N, 3, F, dtype=torch.float64)
    if states is not None:
        states.append((s, v))
    for t in range(T):
        p_ = f"L{t}."
        phi = silu(s @ W[p_ + "Wm1"].T + W[p_ + "bm1"]) @ W[p_ + "Wm2"].T + W[p_ + "bm2"]  # [N,3F]
        w = fc[..., None] * (rho @ W[p_ + "Wf"].T + W[p_ + "bf"])                          # [N,N,nS,3F]
        ws, wvs, wvv = w[..., :F], w[..., F:2 * F], w[..., 2 * F:]
        phs, phvs, phvv = phi[:, :F], phi[:, F:2 * F], phi[:, 2 * F:]
        s1 = s + torch.einsum("ijSf,jf->if", ws, phs)
        v1 = v + torch.einsum("ijSf,jf,ijSc->icf", wvs, phvs, u) \
               + torch.einsum("ijSf,jf,jcf->icf", wvv, phvv, v)
        p = v1 @ W[p_ + "U"].T
        q = v1 @ W[p_ + "V"].T
        nrm = torch.sqrt((q * q).sum(1) + eps)
        D = (p * q).sum(1)
        a = silu(torch.cat([s1, nrm], -1) @ W[p_ + "Wu1"].T + W[p_ + "bu1"]) @ W[p_ + "Wu2"].T + W[p_ + "bu2"]
        avv, asv, ass = a[:, :F], a[:, F:2 * F], a[:, 2 * F:]
        v = v1 + avv[:, None, :] * p
        s = s1 + asv * D + ass
        if states is not None:
            states.append((s, v))
    Ei = silu(s @ W["Wr1"].T + W["br1"]) @ W["wr2"] + W["br2"]
    return Ei[:n_local].sum(), Ei


@pytest.mark.parametrize("periodic", [True, False])
def test_dense_autograd_restatement(periodic):
    import torch
    pos, types, box = _small_water()
    blob = _blob(SMALL_MODEL)
    hdr, arrs = gen.parse_blob(blob)
    N = len(pos)
    n_local = N if periodic else N - 9           # open mode: last 9 atoms act as (un-owned) ghosts
    r = oracle.compute(blob, pos, types, box, n_local=n_local, n_ghost=N - n_local, periodic=periodic)
    P = torch.tensor(pos, dtype=torch.float64, requires_grad=True)
    E, Ei = _dense_energy_torch(arrs, hdr, P, types, torch.tensor(box), n_local, periodic)
    gP, = torch.autograd.grad(E, P)
    assert abs(E.item() - r["energy"]) <= 1e-10 * max(1, abs(r["energy"]))
    np.testing.assert_allclose(Ei.detach().numpy(), r["atom_energy"], rtol=0, atol=1e-10)
    np.testing.assert_allclose(-gP.numpy(), r["forces"], rtol=0, atol=1e-9)


@pytest.mark.parametrize("periodic", [True, False])
def test_state_dump_matches_dense_restatement(periodic):
    """Pin of the oracle's `state_dump` export (the reference of every layer-state assertion of the GPU tests):
    [(T+1) x N x 4F] = (s | v_x | v_y | v_z) after the embedding and after each layer, against the per-layer s, v of the
    dense restatement.  A wrong stride, layer offset or component order fails here."""
    import torch
    pos, types, box = _small_water()
    blob = _blob(SMALL_MODEL)
    hdr, arrs = gen.parse_blob(blob)
    N, F, T = len(pos), hdr["F"], hdr["T"]
    n_local = N if periodic else N - 9
    r = oracle.compute(blob, pos, types, box, n_local=n_local, n_ghost=N - n_local, periodic=periodic, want_states=True)
    st = []
    _dense_energy_torch(arrs, hdr, torch.tensor(pos, dtype=torch.float64), types, torch.tensor(box), n_local, periodic, st)
    assert r["states"].shape == (T + 1, N, 4 * F) and len(st) == T + 1
    for t, (s_t, v_t) in enumerate(st):
        np.testing.assert_allclose(r["states"][t, :, :F], s_t.numpy(), rtol=0, atol=1e-10)
        for c in range(3):
            np.testing.assert_allclose(r["states"][t, :, (1 + c) * F:(2 + c) * F], v_t[:, c, :].numpy(), rtol=0, atol=1e-10)
    assert np.abs(r["states"][0, :, F:]).max() == 0.0            # v^0 = 0
    assert np.abs(r["states"][T, :, F:]).max() > 0.0             # and the vector channels are not all zero later


def test_dense_autograd_virial_open_mode():
    """W_ab = -dE/d(eps_ab) under a homogeneous strain of all positions (open boundaries, any eps)."""
    import torch
    pos, types, box = _small_water()
    blob = _blob(SMALL_MODEL)
    hdr, arrs = gen.parse_blob(blob)
    N = len(pos)
    r = oracle.compute(blob, pos, types, box, n_local=N - 5, n_ghost=5, periodic=False)
    P = torch.tensor(pos, dtype=torch.float64)
    eps_ = torch.zeros(3, 3, dtype=torch.float64, requires_grad=True)
    E, _ = _dense_energy_torch(arrs, hdr, P @ (torch.eye(3, dtype=torch.float64) + eps_).T, types,
                               torch.tensor(box), N - 5, False)
    gE, = torch.autograd.grad(E, eps_)
    np.testing.assert_allclose(-gE.numpy(), r["virial9"], rtol=0, atol=1e-9)


# ------------------------------------------------------------------ invariances
def _rand_rotation(rng, reflect=False):
    q, _ = np.linalg.qr(rng.standard_normal((3, 3)))
    if (np.linalg.det(q) < 0) != reflect:
        q[:, 0] *= -1
    return q


def test_translation_invariance_periodic(cfg1):
    c = cfg1
    r0 = oracle.compute(c["blob"], c["pos"], c["types"], c["box"])
    shift = np.array([3.3, -1.7, 0.9])
    r1 = oracle.compute(c["blob"], c["pos"] + shift, c["types"], c["box"])       # un-wrapped on purpose
    assert abs(r0["energy"] - r1["energy"]) < 1e-9
    np.testing.assert_allclose(r0["forces"], r1["forces"], atol=1e-9)
    np.testing.assert_allclose(r0["virial"], r1["virial"], atol=1e-8)
    assert r0["n_edges"] == r1["n_edges"]


@pytest.mark.parametrize("reflect", [False, True])
def test_rotation_equivariance_open_cluster(reflect):
    rng = np.random.default_rng(3)
    pos, types, box = _small_water(n_mol=25, L=11.0)
    blob = _blob(SMALL_MODEL)
    N = len(pos)
    Rm = _rand_rotation(rng, reflect)
    r0 = oracle.compute(blob, pos, types, box, n_local=N - 6, n_ghost=6, periodic=False)
    r1 = oracle.compute(blob, pos @ Rm.T + 5.0, types, box, n_local=N - 6, n_ghost=6, periodic=False)
    assert abs(r0["energy"] - r1["energy"]) < 1e-10
    np.testing.assert_allclose(r0["forces"] @ Rm.T, r1["forces"], atol=1e-10)
    np.testing.assert_allclose(Rm @ r0["virial9"] @ Rm.T, r1["virial9"], atol=1e-9)


def test_axis_permutation_and_mirror_periodic():
    """Periodic boxes only admit the cubic point group: permute axes (with an orthorhombic box) + mirror x."""
    box = np.array([10.2, 11.1, 12.3])
    pos, types = gen.water_box(22, box, 5)
    blob = _blob(SMALL_MODEL)
    r0 = oracle.compute(blob, pos, types, box)
    perm = [2, 0, 1]
    pos1 = pos[:, perm].copy(); box1 = box[perm].copy()
    pos1[:, 0] = box1[0] - pos1[:, 0]
    r1 = oracle.compute(blob, pos1, types, box1)
    f0 = r0["forces"][:, perm].copy(); f0[:, 0] *= -1
    assert abs(r0["energy"] - r1["energy"]) < 1e-10
    np.testing.assert_allclose(f0, r1["forces"], atol=1e-10)


def test_atom_permutation(cfg1):
    c = cfg1
    rng = np.random.default_rng(0)
    perm = rng.permutation(len(c["pos"]))
    r0 = oracle.compute(c["blob"], c["pos"], c["types"], c["box"])
    r1 = oracle.compute(c["blob"], c["pos"][perm], c["types"][perm], c["box"])
    assert abs(r0["energy"] - r1["energy"]) < 1e-9
    np.testing.assert_allclose(r0["forces"][perm], r1["forces"], atol=1e-9)


def test_newton_third_law_and_virial_symmetry(cfg1):
    c = cfg1
    r = oracle.compute(c["blob"], c["pos"], c["types"], c["box"])
    assert np.abs(r["forces"].sum(0)).max() < 1e-10
    W = r["virial9"]
    assert np.abs(W - W.T).max() < 1e-9 * np.abs(W).max()


def test_virial_is_strain_derivative_periodic(cfg1):
    """W_ab = -dE/d(eps_ab): central differences of E under a homogeneous strain of box AND positions
    (diagonal strains keep the box orthorhombic; shear is covered by the open-mode autograd test)."""
    c = cfg1
    r = oracle.compute(c["blob"], c["pos"], c["types"], c["box"])
    h = 1e-5
    for a in range(3):
        e = []
        for k in (1, -1, 2, -2):
            sc = np.ones(3); sc[a] += k * h
            e.append(oracle.compute(c["blob"], c["pos"] * sc, c["types"], c["box"] * sc)["energy"])
        dE = (8 * (e[0] - e[1]) - (e[2] - e[3])) / (12 * h)
        assert abs(-dE - r["virial"][a]) < 1e-5 * abs(r["virial"][a]) + 1e-6, (a, -dE, r["virial"][a])


def test_extensivity_2x2x2(cfg1):
    c = cfg1
    r1 = oracle.compute(c["blob"], c["pos"], c["types"], c["box"])
    p8, t8, b8 = gen.replicate(c["pos"], c["types"], c["box"])
    r8 = oracle.compute(c["blob"], p8, t8, b8)
    assert abs(r8["energy"] - 8 * r1["energy"]) <= 1e-9 * abs(8 * r1["energy"])
    np.testing.assert_allclose(r8["forces"], np.tile(r1["forces"], (8, 1)), atol=1e-9)
    np.testing.assert_allclose(r8["virial"], 8 * r1["virial"], rtol=1e-9)
    assert r8["n_edges"] == 8 * r1["n_edges"]


def test_ghost_images_reproduce_periodic(cfg1):
    """Halo T*rc = 10 A of periodic images passed as ghosts (+ owner fold) == periodic result
    (each U_i computed once on a complete environment; partial forces summed, :64-66)."""
    c = cfg1
    m = c["model"]
    r0 = oracle.compute(c["blob"], c["pos"], c["types"], c["box"])
    gpos, gown, _ = gen.periodic_ghosts(c["pos"], c["box"], m["T"] * m["rc"])
    pos = np.concatenate([c["pos"], gpos]); types = np.concatenate([c["types"], c["types"][gown]])
    r1 = oracle.compute(c["blob"], pos, types, c["box"], n_local=len(c["pos"]), n_ghost=len(gpos), ghost_owner=gown)
    assert abs(r0["energy"] - r1["energy"]) < 1e-9
    np.testing.assert_allclose(r1["forces"][:len(c["pos"])], r0["forces"], atol=1e-9)
    assert np.abs(r1["forces"][len(c["pos"]):]).max() == 0.0
    np.testing.assert_allclose(r1["virial"], r0["virial"], rtol=1e-9, atol=1e-8)
    # without the owner map the partial forces stay on the ghost rows (LAMMPS reverse-comm convention)
    r2 = oracle.compute(c["blob"], pos, types, c["box"], n_local=len(c["pos"]), n_ghost=len(gpos))
    folded = r2["forces"][:len(c["pos"])].copy()
    np.add.at(folded, gown, r2["forces"][len(c["pos"]):])
    np.testing.assert_allclose(folded, r0["forces"], atol=1e-9)
    # a 1*rc halo (config 3 as specified, reading A18) is a truncated graph: NOT the periodic result
    gpos5, gown5, _ = gen.periodic_ghosts(c["pos"], c["box"], m["rc"])
    pos5 = np.concatenate([c["pos"], gpos5]); types5 = np.concatenate([c["types"], c["types"][gown5]])
    r5 = oracle.compute(c["blob"], pos5, types5, c["box"], n_local=len(c["pos"]), n_ghost=len(gpos5), ghost_owner=gown5)
    assert abs(r5["energy"] - r0["energy"]) > 1e-6


# ------------------------------------------------------------------ closed forms
def _silu(x):
    return x / (1 + np.exp(-x))


def test_no_message_model_gives_species_energies(cfg1):
    """Wm2 = 0, bm2 = 0 -> phi = 0 -> no messages: F == 0 and E = sum_species count * e_species, where
    e_species follows from T applications of the update with v' = 0 (p = q = 0, n = sqrt(eps), D = 0)."""
    c = cfg1
    m = c["model"]
    F, T = m["F"], m["T"]
    over = {}
    for t in range(T):
        over[f"L{t}.Wm2"] = np.zeros((3 * F, F)); over[f"L{t}.bm2"] = np.zeros(3 * F)
    blob = _blob(m, overrides=over)
    hdr, A = gen.parse_blob(blob)
    r = oracle.compute(blob, c["pos"], c["types"], c["box"])
    assert np.abs(r["forces"]).max() == 0.0 and np.abs(r["virial"]).max() == 0.0
    e_species = []
    for z in range(m["n_species"]):
        s = A["Emb"][z].copy()
        for t in range(T):
            sn = np.concatenate([s, np.full(F, np.sqrt(hdr["eps"]))])
            a = A[f"L{t}.Wu2"] @ _silu(A[f"L{t}.Wu1"] @ sn + A[f"L{t}.bu1"]) + A[f"L{t}.bu2"]
            s = s + a[2 * F:]
        e_species.append(A["wr2"] @ _silu(A["Wr1"] @ s + A["br1"]) + A["br2"][0])
    counts = np.bincount(c["types"], minlength=m["n_species"])
    assert abs(r["energy"] - counts @ np.array(e_species)) < 1e-10


def test_dimer_radial_force_and_virial():
    """Dimer in a large box: E = E(d); F = -/+ (dE/dd) u; W = -d (dE/dd) u(x)u."""
    model = dict(n_species=2, F=8, K=6, T=2, rc=5.0, wseed=5)
    blob = _blob(model)
    box = np.full(3, 30.0)
    u = np.array([1.0, 2.0, -2.0]) / 3.0
    types = np.array([0, 1], np.int32)

    def run(d):
        pos = np.array([[10.0, 10.0, 10.0], [10.0, 10.0, 10.0] + d * u])
        return oracle.compute(blob, pos, types, box)

    d, h = 2.3, 1e-4
    r = run(d)
    dE = (8 * (run(d + h)["energy"] - run(d - h)["energy"]) - (run(d + 2 * h)["energy"] - run(d - 2 * h)["energy"])) / (12 * h)
    np.testing.assert_allclose(r["forces"][1], -dE * u, atol=1e-8)
    np.testing.assert_allclose(r["forces"][0], +dE * u, atol=1e-8)
    np.testing.assert_allclose(r["virial9"], -d * dE * np.outer(u, u), atol=1e-7)
    # rotating the dimer axis leaves E unchanged
    assert r["n_edges"] == 2


def test_energy_continuous_across_cutoff():
    """rho_n(rc) = 0 and fc(rc) = 0: E is continuous when a pair crosses rc (and equals the isolated sum)."""
    model = dict(n_species=2, F=8, K=6, T=2, rc=5.0, wseed=5)
    blob = _blob(model)
    box = np.full(3, 30.0)
    types = np.array([0, 1], np.int32)

    def run(d):
        return oracle.compute(blob, np.array([[5.0, 5.0, 5.0], [5.0 + d, 5.0, 5.0]]), types, box)

    inside, outside, far = run(5.0 - 1e-9), run(5.0 + 1e-9), run(9.0)
    assert inside["n_edges"] == 2 and outside["n_edges"] == 0
    assert abs(inside["energy"] - outside["energy"]) < 1e-12 * 1e3
    assert outside["energy"] == far["energy"]
    assert np.abs(inside["forces"]).max() < 1e-6          # fc'(rc) = 0, rho_n(rc) = 0: force vanishes too


# ------------------------------------------------------------------ neighbour set
def test_neighbors_match_kdtree_and_are_symmetric(cfg1):
    from scipy.spatial import cKDTree
    c = cfg1
    i, j, S = oracle.neighbors(c["pos"], c["box"], 5.0)
    # library routine: periodic KD-tree pairs (unordered, i<j); L >= 2 rc so each pair has one image
    pairs = cKDTree(c["pos"], boxsize=c["box"]).query_pairs(5.0, output_type="ndarray")
    want = set(map(tuple, pairs)) | set(map(tuple, pairs[:, ::-1]))
    got = set(zip(i.tolist(), j.tolist()))
    assert len(got) == len(i)            # one image per ordered pair
    assert got == want
    trip = set(zip(i.tolist(), j.tolist(), map(tuple, S.tolist())))
    assert all((b, a, (-s[0], -s[1], -s[2])) in trip for a, b, s in trip)
    # image is the one that realises the distance
    r = c["pos"][j] + S * c["box"] - c["pos"][i]
    assert ((r * r).sum(1) < 25.0).all()


def test_perfect_diamond_has_28_neighbours():
    pos, types, box = gen.diamond(3, 5.43, 0.0, 0)           # 216 atoms, L = 16.29 >= 2 rc
    i, j, S = oracle.neighbors(pos, box, 5.0)
    assert (np.bincount(i, minlength=len(pos)) == 28).all()


def test_liquid_density_gives_about_52_neighbours():
    c = gen.make_config(2, n_mol=1000, L=31.04)
    i, _, _ = oracle.neighbors(c["pos"], c["box"], 5.0)
    nbar = len(i) / len(c["pos"])
    expect = 4.0 / 3.0 * np.pi * 125.0 * len(c["pos"]) / c["box"].prod()
    assert abs(nbar - expect) < 0.05 * expect, (nbar, expect)


def test_unwrapped_positions_need_wider_image_range():
    """Positions up to one box length outside [0, L): the definition with S in {-2..2}^3 still finds the
    same graph (images re-labelled), reading A13."""
    box = np.array([10.5, 10.5, 10.5])
    pos, types = gen.water_box(15, box, 9)
    rng = np.random.default_rng(1)
    shift = rng.integers(-1, 2, size=pos.shape) * box
    i0, j0, S0 = oracle.neighbors(pos, box, 5.0, smax=1)
    i1, j1, S1 = oracle.neighbors(pos + shift, box, 5.0, smax=3)
    assert len(i0) == len(i1)
    w = shift / box
    a = set(zip(i0.tolist(), j0.tolist(), map(tuple, S0.tolist())))
    b = set(zip(i1.tolist(), j1.tolist(), map(tuple, (S1 + (w[j1] - w[i1])).astype(int).tolist())))
    assert a == b


def test_block_decomposition_of_the_fullsize_goldens_is_exact(cfg1, tmp_path):
    """tests/golden/make_golden_fullsize.py sums the oracle over blocks of local atoms with a T * rc halo of ghosts
    (PAPER.md:58, 64-66).  On config 1 (box 12.42 A < halo: up to 27 + images of an atom inside one block's halo) the
    2 x 2 x 2 block sum must reproduce the periodic whole-system oracle: E, the virial and every force."""
    import importlib.util
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "make_golden_fullsize.py")
    spec = importlib.util.spec_from_file_location("make_golden_fullsize", path)
    G = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(G)
    E, W6, F = G.run(1, 2, 10.0, 8, str(tmp_path / "g.json"), log=lambda s: None)     # T rc = 10 A for the 2-layer model
    ref = oracle.compute(cfg1["blob"], cfg1["pos"], cfg1["types"], cfg1["box"])
    assert abs(E - ref["energy"]) <= 1e-10 * abs(ref["energy"])
    np.testing.assert_allclose(W6, ref["virial"], rtol=0, atol=1e-9 * np.abs(ref["virial"]).max())
    np.testing.assert_allclose(F, ref["forces"], rtol=0, atol=1e-9 * np.abs(ref["forces"]).max())
    import json
    doc = json.load(open(tmp_path / "g.json"))
    assert doc["energy"] == E and len(doc["sample_idx"]) == 8 and doc["meta"]["blocks"] == [2, 2, 2]


def test_oracle_reproduces_golden_config1():
    """Regression guard for the oracle itself (tests/golden/oracle_config1.txt, written by tests/golden/make_golden.py from
    oracle/ only): a change of its arithmetic has to be deliberate -- re-run the script and justify it in the commit."""
    import importlib.util
    import os
    here = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(here, "make_golden.py"))
    mg = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mg)
    c, r = mg.evaluate()
    want = {}
    for line in open(os.path.join(here, "oracle_config1.txt")):
        if line.startswith("#"):
            continue
        k, *v = line.split()
        if k == "force":
            want.setdefault("force", {})[int(v[0])] = np.array([float(x) for x in v[1:]])
        else:
            want[k] = np.array([float(x) for x in v])
    assert len(c["pos"]) == int(want["n_atoms"][0]) and int(r["n_edges"]) == int(want["n_edges"][0])
    # fp64 results depend on the BLAS summation order (thread count): 1e-10 relative, far below any tolerance of the path
    assert abs(float(r["energy"]) - want["energy"][0]) <= 1e-10 * abs(want["energy"][0])
    assert np.abs(np.asarray(r["virial"]).ravel() - want["virial"]).max() <= 1e-9 * np.abs(want["virial"]).max()
    frms = np.sqrt((r["forces"] ** 2).mean())
    for a, f in want["force"].items():
        assert np.abs(r["forces"][a] - f).max() <= 1e-9 * frms
