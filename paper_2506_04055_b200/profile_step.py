"""Run a few steps of one BASELINE.json config through the C ABI (device-resident inputs) -- the short command that
the ncu captures under profiles/ wrap:

    python -m paper_2506_04055_b200.profile_step <config 1-5> <steps> [option=value ...]

Options are passed to mlp_set_option (e.g. edge_path=1, gemm_fwd_tc=1).  The full-size workload is generated once and
cached under /tmp (same cache as bench.py).
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def main():
    import torch
    import bench
    import paper_2506_04055_b200 as P
    k, steps = int(sys.argv[1]), int(sys.argv[2])
    c, blob = bench._cached_workload(k)
    m = c["model"]
    dev = torch.device("cuda:0")
    M = P.Model(blob, m["n_species"], m["rc"], len(c["pos"]))
    for a in sys.argv[3:]:
        n, v = a.split("=")
        M.set_option(n, int(v))
    pos = torch.from_numpy(c["pos"]).to(dev)
    types = torch.from_numpy(c["types"]).to(dev)
    go = None if c["ghost_owner"] is None else torch.from_numpy(np.ascontiguousarray(c["ghost_owner"], np.int32)).to(dev)
    for _ in range(steps):
        e, f, w = M.compute(pos, types, c["box"], c["n_local"], c["n_ghost"], go)
    torch.cuda.synchronize()
    print("E", float(e[0]), M.stats())


if __name__ == "__main__":
    main()
