#!/usr/bin/env python
"""Full-size oracle goldens for BASELINE.json configs 2-5: total energy, virial and a stratified force sample.

    python tests/golden/make_golden_fullsize.py --config 5 [--blocks 4] [--out tests/golden/fullsize_config5.json]

Calls ONLY gen/ (seeded inputs) and oracle/ (fp64 CPU oracle).  Nothing here touches the CUDA path.

Why blocks are exact ("each U_i ... computed exactly once ... on a sub-graph with complete
environment"; partial forces of all copies are summed): the model is semi-local with receptive
field T * rc.  The box is tiled into bx * by * bz blocks; the atoms of one block are passed to the oracle as LOCAL
atoms and every atom (or periodic image of an atom) within `halo` >= T * rc of the block as a GHOST, with open
boundaries and no owner map -- exactly the local + ghost contract of the C ABI.  Then

    E   = sum over blocks of  E_block              (E_block = sum of E_i over the block's local atoms)
    W   = sum over blocks of  W_block              (W_block = -dE_block/d(strain): the oracle's ghost-mode virial over
                                                    all edges of the block's sub-graph)
    F_k = sum over blocks of  (partial force of E_block on every copy of atom k in that block's sub-graph)

are the whole-system values: every E_i appears in exactly one block with its complete T-hop environment, and the
gradient of a sum is the sum of the gradients.  The ghost == periodic pin of tests/test_oracle_pins.py covers this
use of the oracle.  For config 3 (already a local + ghost system with open boundaries) the blocks tile the bounding
box of all atoms, the original ghosts never become block-locals (their E_i is not part of E), and partial forces
are kept per given row (no owner fold), matching mlp_compute(ghost_owner = NULL).

The stored sample (>= 64 atoms per stratum where the stratum exists) holds indices and fp64 forces; F_rms over all
local atoms is stored as well, so a test can evaluate both force criteria of north_star on the sample.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)

import gen  # noqa: E402
import oracle  # noqa: E402


def _images(pos, box, lo, hi, halo, periodic):
    """Indices + shifted positions of all atoms / periodic images inside [lo - halo, hi + halo) (excluding nothing)."""
    out_i, out_p = [], []
    rng = []
    for d in range(3):
        if periodic:
            smin = int(np.floor((lo[d] - halo) / box[d]))
            smax = int(np.floor((hi[d] + halo) / box[d]))
            rng.append(range(smin, smax + 1))        # image shifts S for which pos + S * box can fall in the window
        else:
            rng.append(range(0, 1))
    idx = np.arange(len(pos))
    for sx in rng[0]:
        for sy in rng[1]:
            for sz in rng[2]:
                p = pos + np.array([sx, sy, sz]) * box
                m = np.all((p >= lo - halo) & (p < hi + halo), axis=1)
                if m.any():
                    out_i.append(idx[m]); out_p.append(p[m])
    return np.concatenate(out_i), np.concatenate(out_p)


def run(k, blocks, halo, n_sample, out, log=print):
    c = gen.make_config(k)
    mdl = c["model"]
    blob = gen.make_weights(mdl["n_species"], mdl["F"], mdl["K"], mdl["T"], mdl["rc"], seed=mdl["wseed"])
    assert halo >= mdl["T"] * mdl["rc"], "halo must cover the receptive field T * rc (PAPER.md:58)"
    pos, types, box = c["pos"], c["types"], np.asarray(c["box"], np.float64)
    N, nl = len(pos), c["n_local"]
    periodic = c["n_ghost"] == 0
    if periodic:
        glo, ghi = np.zeros(3), box.copy()
    else:
        glo, ghi = pos.min(0) - 1e-6, pos.max(0) + 1e-6
    is_local = np.arange(N) < nl
    E, W9 = 0.0, np.zeros((3, 3))
    Fsum = np.zeros((N, 3))
    t_start = time.time()
    nb = [blocks] * 3 if isinstance(blocks, int) else list(blocks)
    edges = [np.linspace(glo[d], ghi[d], nb[d] + 1) for d in range(3)]
    done = 0
    covered = np.zeros(N, bool)
    for bx in range(nb[0]):
        for by in range(nb[1]):
            for bz in range(nb[2]):
                lo = np.array([edges[0][bx], edges[1][by], edges[2][bz]])
                hi = np.array([edges[0][bx + 1], edges[1][by + 1], edges[2][bz + 1]])
                idx, p = _images(pos, box, lo, hi, halo, periodic)
                inside = np.all((p >= lo) & (p < hi), axis=1) & is_local[idx]
                loc = np.nonzero(inside)[0]
                if len(loc) == 0:
                    done += 1
                    continue
                assert not covered[idx[loc]].any()
                covered[idx[loc]] = True
                gh = np.nonzero(~inside)[0]
                order = np.concatenate([loc, gh])
                bp = p[order] - (lo - halo) + 1.0                   # open boundaries: any rigid shift is allowed
                t0 = time.time()
                r = oracle.compute(blob, bp, types[idx[order]], np.array([1e4, 1e4, 1e4]), n_local=len(loc),
                                   n_ghost=len(gh), periodic=False)
                E += r["energy"]
                W9 += r["virial9"]
                np.add.at(Fsum, idx[order], r["forces"])
                done += 1
                log(f"config {k}: block {done}/{nb[0] * nb[1] * nb[2]}  local {len(loc)}  total {len(order)}  "
                    f"{time.time() - t0:.1f} s  (elapsed {time.time() - t_start:.0f} s)")
    assert covered[:nl].all() and not covered[nl:].any()
    W6 = np.array([W9[0, 0], W9[1, 1], W9[2, 2], 0.5 * (W9[0, 1] + W9[1, 0]), 0.5 * (W9[0, 2] + W9[2, 0]),
                   0.5 * (W9[1, 2] + W9[2, 1])])
    frms = float(np.sqrt((Fsum[:nl] ** 2).mean()))
    # stratified sample: bulk / interface (slab surface) / next to the ghost halo / ghosts / chain atoms -- where they exist
    rng = np.random.default_rng(20250600 + k)
    strata = {"bulk": np.arange(nl)}
    if k == 3:
        z = pos[:nl, 2]
        strata["surface"] = np.nonzero(z > z.max() - 3.0)[0]
        strata["halo_owner"] = np.unique(np.asarray(c["ghost_owner"], np.int64))
        strata["ghost"] = np.arange(nl, N)
    if k == 5:
        strata["chain"] = np.nonzero(~np.isin(types, (0, 3)))[0]        # C, N, S only occur in the chains
    sample, labels = [], []
    for name, pool in strata.items():
        pick = rng.choice(pool, size=min(n_sample, len(pool)), replace=False)
        sample.append(np.sort(pick)); labels += [name] * len(pick)
    sample = np.concatenate(sample)
    try:
        git = subprocess.run(["git", "-C", ROOT, "rev-parse", "HEAD"], capture_output=True, text=True).stdout.strip()
    except Exception:
        git = "unknown"
    meta = dict(config=k, name=c["name"], n_local=nl, n_total=N, blocks=nb, halo=halo, model=mdl,
                oracle_threads=oracle.threads(), seconds=round(time.time() - t_start, 1), script_git=git,
                box=box.tolist())
    # text fixture: repr() of a Python float round-trips the fp64 value exactly
    doc = dict(meta=meta, energy=float(E), virial=[float(x) for x in W6], virial9=[[float(x) for x in r] for r in W9],
               f_rms=frms, f_sum=[float(x) for x in Fsum[:nl].sum(0)],
               sample_idx=[int(i) for i in sample], sample_strata=labels,
               sample_forces=[[float(x) for x in Fsum[i]] for i in sample])
    with open(out, "w") as fh:
        json.dump(doc, fh, indent=0)
        fh.write("\n")
    log(f"config {k}: E = {E!r}  E/atom = {E / nl!r}  F_rms = {frms!r}  -> {out}  ({meta['seconds']} s)")
    return E, W6, Fsum


if __name__ == "__main__":
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, required=True, choices=(1, 2, 3, 4, 5))
    ap.add_argument("--blocks", type=int, nargs="+", default=None, help="blocks per dimension (1 or 3 numbers)")
    ap.add_argument("--halo", type=float, default=15.0)
    ap.add_argument("--sample", type=int, default=96, help="atoms per stratum")
    ap.add_argument("--out", default=None)
    a = ap.parse_args()
    blocks = a.blocks or {1: [1], 2: [2], 3: [3, 3, 3], 4: [4], 5: [5]}[a.config]
    blocks = blocks[0] if len(blocks) == 1 else blocks
    out = a.out or os.path.join(HERE, f"fullsize_config{a.config}.json")
    run(a.config, blocks, a.halo, a.sample, out, log=lambda s: print(s, flush=True))
