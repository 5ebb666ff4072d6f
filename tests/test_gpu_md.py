"""The path as an MD engine calls it: the paper's own PaiNN shapes (4 layers, F = 64 and
128) against the oracle, alternative implementations of the same arithmetic (mlp_set_option switches) against
the oracle, and a short NVE trajectory driven by the GPU forces whose total energy must be conserved (PAPER.md:232, 252-254
run NVT / NVE production steps; here 100 velocity-Verlet steps with unit masses).  Energy conservation ties E and F of the
CUDA path to each other independently of the oracle: F must be the exact gradient of the E that is returned.
"""
import numpy as np
import pytest

import gen
from test_gpu_parity import _blob, _check, _gpu_eval, _oracle_eval, _same_edges, _torch

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("F", [64, 128])
def test_paper_shapes_four_layers(F):
    c = gen.make_config(2, n_mol=500, L=24.64, T=4, F=F)
    blob = _blob(c["model"])
    m, e, f, w = _gpu_eval(c, blob)
    ne = _same_edges(m, c)
    ref = _oracle_eval(c, blob)
    assert ref["n_edges"] == ne
    _check(c, e, f, w, ref, f"config 2 recipe, PaiNN 4 x {F} (N={len(c['pos'])}, E={ne})")


@pytest.mark.parametrize("opts", [dict(edge_path=1), dict(gemm_fwd_exact=0), dict(gemm_bwd_exact=1),
                                  dict(l0_collapse=0), dict(atoms_per_unit=5), dict(atoms_per_unit=31), dict(cell_strip=0), dict(cell_strip=1), dict(cell_strip=4)])
def test_alternative_kernel_paths_match_oracle(opts):
    """Every switch of mlp_set_option selects another implementation of the same arithmetic; each must meet the same
    tolerances (the plain fp32 edge kernels, the fp32 FFMA forward GEMM, the exact-slice adjoint GEMM, the per-edge layer-0
    kernels, other work-unit sizes and cell orders).  Options belong to the model they are set on."""
    import paper_2506_04055_b200 as P
    torch = _torch()
    c = gen.make_config(5, n_slots=1200, L=32.98)
    blob = _blob(c["model"])
    dev = torch.device("cuda:0")
    with P.Model(blob, c["model"]["n_species"], c["model"]["rc"], len(c["pos"])) as m:
        for k, v in opts.items():
            m.set_option(k, v)
        e, f, w = m.compute(torch.from_numpy(c["pos"]).to(dev), torch.from_numpy(c["types"]).to(dev), c["box"])
        torch.cuda.synchronize()
        e, f, w = float(e[0]), f.cpu().numpy(), w.cpu().numpy()
    ref = _oracle_eval(c, blob)
    _check(c, e, f, w, ref, f"config 5 recipe reduced, options {opts}")


@pytest.mark.parametrize("k,over", [(1, {}), (2, dict(n_mol=300, L=20.78))])
def test_nve_energy_conservation(k, over):
    import paper_2506_04055_b200 as P
    torch = _torch()
    c = gen.make_config(k, **over)
    blob = _blob(c["model"])
    dev = torch.device("cuda:0")
    N = len(c["pos"])
    box = np.asarray(c["box"], np.float64)
    types = torch.from_numpy(c["types"]).to(dev)
    with P.Model(blob, c["model"]["n_species"], c["model"]["rc"], N) as m:
        def ef(x):
            e, f, _ = m.compute(torch.from_numpy(np.ascontiguousarray(x)).to(dev), types, box)
            torch.cuda.synchronize()
            return float(e[0]), f.cpu().numpy()

        x = c["pos"].copy()
        e0, f = ef(x)
        frms = np.sqrt((f ** 2).mean())
        # time step: ~0.0125 A of ballistic travel over 100 steps from rest under the initial forces (unit masses).  The
        # random-weight potential has no repulsive core and is unbounded below, so long trajectories run away (atoms
        # accelerate into ever steeper regions); 100 short steps stay where the dynamics is well resolved
        dt = np.sqrt(2.5e-6 / frms)
        v = np.zeros_like(x)
        etot, ke_max = [e0], 0.0
        for step in range(100):
            v += 0.5 * dt * f
            x += dt * v                      # positions are NOT wrapped: the library wraps internally (reading A13)
            e, f = ef(x)
            v += 0.5 * dt * f
            ke = 0.5 * float((v * v).sum())
            ke_max = max(ke_max, ke)
            etot.append(e + ke)
    etot = np.asarray(etot)
    drift = np.abs(etot - etot[0]).max()
    print(f"config {k}: N={N} dt={dt:.3e} KE_max={ke_max:.4e} max|dE_tot|={drift:.3e} ratio={drift / ke_max:.2e}")
    assert ke_max > 0 and np.isfinite(etot).all()
    # velocity Verlet conserves E up to O(dt^2) oscillations; the bound also covers the fp32 noise of E (1e-4 per atom)
    assert drift <= 2e-3 * ke_max + 2e-4 * N, (drift, ke_max)
