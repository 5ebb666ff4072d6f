#!/usr/bin/env python
"""bench.py -- atom-steps/s of the PaiNN E + F + virial hot path (BASELINE.json metric) on synthetic workloads.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 5] [--impl ours|reference]

One "step" = one full mlp_compute (neighbour rebuild + forward + adjoint + force/virial assembly) over the
whole system.  N > 1 (torchrun): the path does not shard inside one evaluation (BASELINE.json: one GPU, no
collectives), so every rank evaluates its own replica of the workload ("weak" scaling, no data-path collective);
value = N * n_local / max-over-ranks time.  Prints ONE JSON line on rank 0.
--impl reference times the fp64 CPU oracle (oracle/) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import gen  # noqa: E402

METRIC = "atom-steps/s (E+F+virial) PaiNN F=128 at 1M atoms"
UNIT = "atom-steps/s"
# bounded CPU-oracle sample: reduced replica of the same recipe (O(N^2) neighbour search keeps it small)
CPU_SAMPLE = {5: dict(n_slots=6000, L=56.41), 4: dict(ncell=9), 2: dict(n_mol=2400, L=41.55), 1: {},
              3: dict(n_mol=1500, L=35.56)}


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm=d["hbm_gbs"], bf16=d["bf16_tflops"], bf16_sus=d["bf16_tflops_sustained"],
                    sm_max=d.get("sm_max_mhz", 1965.0), src="measured")
    return dict(hbm=6650.0, bf16=1590.0, bf16_sus=1400.0, sm_max=1965.0, src="fallback")


def _workload(k, small=False):
    over = {}
    if small:
        over = CPU_SAMPLE[k]
    c = gen.make_config(k, **over)
    m = c["model"]
    blob = gen.make_weights(m["n_species"], m["F"], m["K"], m["T"], m["rc"], seed=m["wseed"])
    return c, blob


def _cached_workload(k):
    """Full-size generation takes a minute (pure-numpy rejection sampling); cache it under /tmp per process tree."""
    path = f"/tmp/painn_b200_cfg{k}.npz"
    if os.path.exists(path):
        try:
            z = np.load(path, allow_pickle=False)
            c = dict(pos=z["pos"], types=z["types"], box=z["box"], n_local=int(z["n_local"]), n_ghost=int(z["n_ghost"]),
                     ghost_owner=z["ghost_owner"] if z["ghost_owner"].size else None, name=str(z["name"]),
                     model=json.loads(str(z["model"])))
            m = c["model"]
            return c, gen.make_weights(m["n_species"], m["F"], m["K"], m["T"], m["rc"], seed=m["wseed"])
        except Exception:
            pass
    c, blob = _workload(k)
    try:
        tmp = path + f".{os.getpid()}.npz"
        np.savez(tmp, pos=c["pos"], types=c["types"], box=c["box"], n_local=c["n_local"], n_ghost=c["n_ghost"],
                 ghost_owner=c["ghost_owner"] if c["ghost_owner"] is not None else np.empty(0, np.int32),
                 name=c["name"], model=json.dumps(c["model"]))
        os.replace(tmp, path)
    except Exception:
        pass
    return c, blob


def _cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except Exception:
        pass
    return "unknown"


def _oracle_time(k, steps, warmup):
    """The fp64 oracle, as it stands, on a bounded reduced sample of config k: the O(N^2) neighbour
    search and the whole evaluation are timed separately, median of `steps` runs each; model = evaluation - search."""
    import oracle
    c, blob = _workload(k, small=True)
    rc = c["model"]["rc"]
    tn, tt = [], []
    for it in range(warmup + steps):
        t0 = time.perf_counter()
        oracle.neighbors(c["pos"], c["box"], rc, periodic=c["n_ghost"] == 0)
        t1 = time.perf_counter()
        oracle.compute(blob, c["pos"], c["types"], c["box"], c["n_local"], c["n_ghost"], c["ghost_owner"])
        t2 = time.perf_counter()
        if it >= warmup:
            tn.append(t1 - t0); tt.append(t2 - t1)
    t, t_n = float(np.median(tt)), float(np.median(tn))
    return dict(value=c["n_local"] / t, unit=UNIT, cores=oracle.threads(), kind="oracle", cpu=_cpu_model(),
                seconds=dict(evaluation=round(t, 3), neighbour_search=round(t_n, 3), model_forward_adjoint=round(max(t - t_n, 0.0), 3)),
                atom_steps_per_s=dict(neighbour_search=c["n_local"] / t_n, model_forward_adjoint=c["n_local"] / max(t - t_n, 1e-9)),
                sample=f"config {k} recipe reduced to {c['n_local']} local atoms ({len(c['pos'])} total), median of "
                       f"{steps} evaluation(s) of {t:.2f} s each (O(N^2) neighbour search {t_n:.2f} s of it; the sample is "
                       f"size-dependent: the search is quadratic)"), t


class _ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-i", str(index), "-lms", "100"], stdout=subprocess.PIPE,
                                      stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.p = None

    def stop(self):
        if self.p is None:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        time.sleep(0.15)
        self.p.terminate()
        try:
            out, _ = self.p.communicate(timeout=5)
        except Exception:
            self.p.kill()
            out = ""
        sm, mx, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.strip().splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return dict(sm_mhz=float(np.median(sm)) if sm else None, sm_max_mhz=max(mx) if mx else None,
                    power_w_max=max(pw) if pw else None, samples=len(sm), reasons=sorted(reasons))


def _stage_work(stats, model, n_atoms, layer0_split=False):
    """Algorithmic work per step of each timed stage: (bound, units, unit-name).
    layer0_split: the collapsed layer-0 passes are timed as their own stage ("layer0"); fwd_edge / bwd_edge then hold
    the T - 1 launches of layers >= 1 only."""
    F, K, T = model["F"], model["K"], model["T"]
    E, N = stats["n_edges"], n_atoms
    R = F // 2
    w = {}
    if layer0_split:
        NP = 128                                       # columns of the per-(receiver, species) radial sums
        # forward: s in, radial sums written and read by the GEMMs, s' / v1 out, one edge record per edge;
        # adjoint: s1b / v1b in, contracted vectors written and read, edge record + reverse index + G read-modify-write
        l0 = N * (F * 4.0 + 2 * 4 * NP * 4.0 + 4 * F * 4.0) + E * 16.0 \
            + N * (4 * F * 4.0 + 2 * 4 * NP * 4.0) + E * (16.0 + 4.0 + 32.0)
        w["layer0"] = ("hbm", l0, "B")
    # edge stages: compulsory HBM bytes (every per-atom row and per-edge record moved once per launch; DESIGN.md
    # section 6).  The kernels are bound by the L2 -> SM row gather (reported separately as roofline.l2_gather), so
    # the HBM fraction states how far that keeps them from the DRAM roof.
    f0 = 0 if layer0_split else 1                      # layer-0 terms of the per-edge kernels (species-table kernels)
    fwd_atom = f0 * (2 * F * 4 + F * 4 + 4 * F * 4) + (T - 1) * (5 * F * 4 + F * 4 + 3 * F * 4 + 4 * F * 4)   # gather rows + residual + outputs
    w["fwd_edge"] = ("hbm", N * float(fwd_atom) + (T - 1 + f0) * E * 16.0, "B")
    bwd_atom = f0 * (4 * F * 4 + 2 * F * 4) + (T - 1) * (4 * F * 4 + 9 * F * 4 + 6 * F * 4)              # gather rows + own rows + sender adjoint
    w["bwd_edge"] = ("hbm", N * float(bwd_atom) + E * (16.0 * (T - 1 + f0) + f0 * 16.0 + 32.0 * (T - 1)), "B")
    # node GEMMs (flop), fwd: phi-MLP F->F->3F, U|V (3 comps) F->2F, update MLP 2F->F->3F ; readout F->R
    fwd = T * N * 2.0 * (F * F + 3 * F * F + 3 * 2 * F * F + 2 * F * F + 3 * F * F) + N * 2.0 * F * R
    w["fwd_node"] = ("tensor", fwd, "flop")
    w["bwd_node"] = ("tensor", fwd, "flop")          # transposed GEMMs only (weights are fixed)
    # neighbour build: read pos (24 B) ~3x, write ej 16 B + img 1 B + rev 4 B per edge
    w["nbr_build"] = ("hbm", N * 24.0 * 3 + E * 21.0, "B")
    # force/virial: G read twice (own + reverse) 16 B, ej 16 B, rev 4 B per edge; forces 24 B per atom
    w["force_virial"] = ("hbm", E * 52.0 + N * 24.0, "B")
    return w


def _max_over_ranks(x, dist, device):
    """Time of the job = the slowest rank's (contract: MAX over ranks); dist is torch.distributed or None (one rank)."""
    import torch
    t = torch.tensor([x], dtype=torch.float64, device=device)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def _job_value(world, n_local, seconds_per_step):
    """Whole-job throughput of `world` independent replicas ("replicas only"): every rank evaluates
    its own n_local atoms per step, nothing is exchanged on the data path."""
    return world * n_local / seconds_per_step


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=5, help="BASELINE.json config (1-5); 5 = 1M-atom headline")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extra", action="store_true", help="skip the list-reuse leg and the small configs 1-3")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    k = args.config

    if args.impl == "reference":
        if rank != 0:
            return 0
        steps = max(1, min(args.steps, 3))
        warm = min(args.warmup, 1)
        cb, t = _oracle_time(k, steps, warm)
        line = dict(impl="reference", metric=METRIC, value=cb["value"], unit=UNIT, n_gpus=args.gpus, steps=steps,
                    warmup=warm, ms_per_step=t * 1e3, higher_is_better=True, scaling="weak", vs_baseline=None,
                    dtype="f64", data="synthetic",
                    config=dict(workload=f"config {k} ({gen.CONFIGS[k]['name']}), bounded CPU sample", sample=cb["sample"]),
                    cpu_baseline=cb, e2e=dict(value=cb["value"], unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0),
                    gpu_launches=0)
        print(json.dumps(line))
        return 0

    import torch
    import paper_2506_04055_b200 as P
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    dev = torch.device(f"cuda:{local_rank}")
    torch.cuda.set_device(dev)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    c, blob = _cached_workload(k)
    model = c["model"]
    N, n_local = len(c["pos"]), c["n_local"]
    m = P.Model(blob, model["n_species"], model["rc"], N)
    # The metric times one FULL mlp_compute, neighbour rebuild included: the Verlet-skin reuse of the
    # library (default on) is switched off for the headline and measured as its own leg below (`list_reuse`).
    m.set_option("skin_mA", 0)
    opts = os.environ.get("PAINN_OPTS", "")          # experiment knobs "name=value,..." (mlp_set_option); default: none
    for kv in filter(None, opts.split(",")):
        name, val = kv.split("=")
        m.set_option(name, int(val))
    pos = torch.from_numpy(c["pos"]).to(dev)
    types = torch.from_numpy(c["types"]).to(dev)
    owner = None if c["ghost_owner"] is None else torch.from_numpy(np.ascontiguousarray(c["ghost_owner"], np.int32)).to(dev)
    out = (torch.empty(1, dtype=torch.float64, device=dev), torch.empty((N, 3), dtype=torch.float64, device=dev),
           torch.empty(6, dtype=torch.float64, device=dev))
    stream = torch.cuda.current_stream(dev)

    def step():
        m.compute(pos, types, c["box"], n_local, c["n_ghost"], owner, out=out, stream=stream)

    def barrier():
        torch.cuda.synchronize(dev)
        if dist is not None:
            dist.barrier()
            torch.cuda.synchronize(dev)

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    # ---- timed region: device-resident inputs, CUDA events on the launching stream ----
    sampler = _ClockSampler(local_rank) if rank == 0 else None
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record(stream)
    for _ in range(args.steps):
        step()
    ev1.record(stream)
    barrier()
    ms_total = ev0.elapsed_time(ev1)
    clocks = sampler.stop() if sampler else None
    stats = m.stats()
    launches = stats["n_launches"] * args.steps
    ms_total = _max_over_ranks(ms_total, dist, dev)
    ms_step = ms_total / args.steps
    value = _job_value(world, n_local, ms_step * 1e-3)

    # ---- per-stage timing (separate pass, not part of `value`) -> roofline of the dominant kernel ----
    m.set_option("stage_timing", 1)
    acc = {}
    reps = max(1, min(args.steps, 5))
    for _ in range(reps):
        step()
        torch.cuda.synchronize(dev)
        for kname, v in m.stage_ms().items():
            acc[kname] = acc.get(kname, 0.0) + v / reps
    m.set_option("stage_timing", 0)
    peaks = _peaks()
    split = acc.get("layer0", 0.0) > 0.0             # collapsed layer-0 passes timed as their own stage
    work = _stage_work(stats, model, N, layer0_split=split)
    T = model["T"]
    n_launch_of = {"fwd_edge": T - 1, "bwd_edge": T - 1} if split else {"fwd_edge": T, "bwd_edge": T}

    def _roof(name):
        bound, units, _ = work[name]
        if bound == "hbm":
            ach, peak, unit = units / (acc[name] * 1e-3) / 1e9, peaks["hbm"], "GB/s"
        elif bound == "tensor":
            # forward: exact fp16 integer-slice kernel, adjoint: 3xTF32; both are rated against the peak of their
            # operand type: fp16 = measured bf16 (sustained, timed inside a long step), tf32 = that x 1.1 / 2.25
            peak = peaks["bf16_sus"] * (1.0 if name == "fwd_node" else 1.1 / 2.25)
            ach, unit = units / (acc[name] * 1e-3) / 1e12, "TFLOP/s"
        else:
            # plain fp32 ALU: 148 SMs x 128 FMA lanes x 2 flop x max SM clock (B200_PROFILING.md nominal table)
            ach, peak, unit = units / (acc[name] * 1e-3) / 1e12, 148 * 128 * 2 * peaks["sm_max"] * 1e6 / 1e12, "TFLOP/s"
        return dict(bound=bound, achieved=ach, peak=peak, unit=unit, frac=ach / peak, ms=round(acc[name], 4))

    stages = {name: _roof(name) for name in acc if name in work}
    dom = max(acc, key=acc.get)
    n_launch = n_launch_of.get(dom, 1)
    dur_ms = acc[dom] / n_launch
    # DRAM bytes per launch of the dominant kernel from the committed ncu capture (profiles/r02_traffic.json, else r01)
    traffic = None
    try:
        tp = os.path.join(ROOT, "profiles", "r02_traffic.json")
        tj = json.load(open(tp if os.path.exists(tp) else os.path.join(ROOT, "profiles", "r01_traffic.json")))
        if k == tj.get("config"):
            traffic = tj["dram_bytes_per_launch"].get(dom)
    except Exception:
        traffic = None
    roofline = dict(kernel=dom, **{kk: stages[dom][kk] for kk in ("bound", "achieved", "peak", "unit", "frac")},
                    traffic=traffic, peak_source=peaks["src"], launches_per_step=n_launch, ms_per_launch=dur_ms,
                    stage_ms={kk: round(v, 4) for kk, v in acc.items()}, stages=stages)
    if dom in ("fwd_edge", "bwd_edge"):
        # the edge kernels are bound by the L2 -> SM row gather, not by DRAM: bytes gathered per edge and channel
        # against the measured gather ceiling of this access pattern (profiles/r01_microbench.md)
        per_edge = {"fwd_edge": 20.0 if split else (8.0 + 20.0 * (T - 1)) / T, "bwd_edge": 16.0}[dom] * model["F"]
        gb = stats["n_edges"] * per_edge / (dur_ms * 1e-3) / 1e9
        # ceiling measured live on this device through the library (mlp_measure_row_gather: 512 B per warp request, rows inside
        # a 400-row window of a 2 GB table, nothing else running); fallback: the round-1 figure of another pod, labelled
        try:
            g_peak, g_src = P.measure_row_gather(2 << 30, 400), "measured in this run (mlp_measure_row_gather, 2 GB table, window 400)"
        except Exception as ex:      # noqa: BLE001
            g_peak, g_src = 16200.0, f"round-1 figure of another pod (profiles/r01_microbench.md); live measurement failed: {ex!r}"
        roofline["l2_gather"] = dict(achieved=gb, peak=g_peak, unit="GB/s", frac=gb / g_peak, peak_source=g_src)
    if split:
        # third view of the edge stages (SURVEY.md 8(d) "edge products + segment sums: plain ALUs"): fp32 instructions the
        # consumers execute per edge and channel (forward 9: 8 FFMA + 1 FMUL; adjoint 21) against the
        # plain-ALU peak = SMs x 128 lanes x max SM clock (B200_PROFILING.md nominal table; one instruction = one lane-op)
        alu_peak = 148 * 128 * peaks["sm_max"] * 1e6 / 1e12
        roofline["alu"] = {}
        for name, per in (("fwd_edge", 9.0), ("bwd_edge", 21.0)):
            if acc.get(name, 0.0) > 0.0:
                ops = stats["n_edges"] * model["F"] * per * (T - 1)
                ach = ops / (acc[name] * 1e-3) / 1e12
                roofline["alu"][name] = dict(achieved=ach, peak=alu_peak, unit="T-op/s (fp32 FMA/MUL lane-ops)", frac=ach / alu_peak,
                                             ops_per_edge_channel=per)

    # ---- end to end through the host-buffer entry point (pinned host memory, copies inside the timed region) ----
    hpos = torch.from_numpy(c["pos"]).pin_memory()
    htypes = torch.from_numpy(c["types"]).pin_memory()
    hown = None if c["ghost_owner"] is None else torch.from_numpy(np.ascontiguousarray(c["ghost_owner"], np.int32)).pin_memory().numpy()
    hout = (torch.empty(1, dtype=torch.float64).pin_memory().numpy(), torch.empty((N, 3), dtype=torch.float64).pin_memory().numpy(),
            torch.empty(6, dtype=torch.float64).pin_memory().numpy())
    e2e_steps = max(1, min(args.steps, 5))
    m.compute_host(hpos.numpy(), htypes.numpy(), c["box"], n_local, c["n_ghost"], hown, out=hout)
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        m.compute_host(hpos.numpy(), htypes.numpy(), c["box"], n_local, c["n_ghost"], hown, out=hout)
    torch.cuda.synchronize(dev)
    te = (time.perf_counter() - t0) / e2e_steps
    te = _max_over_ranks(te, dist, dev)
    e2e = dict(value=_job_value(world, n_local, te), unit=UNIT, ms_per_step=te * 1e3,
               h2d_bytes_per_step=N * 28 + (0 if hown is None else 4 * c["n_ghost"]), d2h_bytes_per_step=N * 24 + 56)

    # ---- the same workload with the kept rc + skin list: static positions, so every step after the
    # first re-filters the list and replays the captured graph -- the steady state of an MD run between rebuilds
    def _time_mode(mm, cc, skin_mA, steps, warm):
        mm.set_option("skin_mA", skin_mA)
        NN = len(cc["pos"])
        p_ = torch.from_numpy(cc["pos"]).to(dev); t_ = torch.from_numpy(cc["types"]).to(dev)
        o_ = None if cc["ghost_owner"] is None else torch.from_numpy(np.ascontiguousarray(cc["ghost_owner"], np.int32)).to(dev)
        out_ = (torch.empty(1, dtype=torch.float64, device=dev), torch.empty((NN, 3), dtype=torch.float64, device=dev),
                torch.empty(6, dtype=torch.float64, device=dev))
        for _ in range(warm):
            mm.compute(p_, t_, cc["box"], cc["n_local"], cc["n_ghost"], o_, out=out_, stream=stream)
        torch.cuda.synchronize(dev)
        a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a0.record(stream)
        for _ in range(steps):
            mm.compute(p_, t_, cc["box"], cc["n_local"], cc["n_ghost"], o_, out=out_, stream=stream)
        a1.record(stream)
        torch.cuda.synchronize(dev)
        return a0.elapsed_time(a1) / steps, mm.stats()

    def _md_protocol(mm, cc, n_equil, n_prod, skin_mA, drift_A):
        """The paper's timing protocol (100 equilibration + 250 production steps, neighbour list with a skin,
        rebuilt when needed) on synthetic motion: the whole configuration drifts rigidly by `drift_A` per step (0.03 A = a
        hydrogen atom at thermal speed, 300 K, 1 fs), so every pair distance -- hence E, F, W -- stays put while the
        displacement test fires after skin / 2 / drift steps: reuse steps replay the captured graph, rebuild steps run the
        cell list; positions leave the box and are wrapped by the library.  (Forces of the random-weight models are not
        physical: integrating them would say nothing about a real run's rebuild cadence.)"""
        mm.set_option("skin_mA", skin_mA)
        NN = len(cc["pos"])
        p_ = torch.from_numpy(cc["pos"]).to(dev); t_ = torch.from_numpy(cc["types"]).to(dev)
        o_ = None if cc["ghost_owner"] is None else torch.from_numpy(np.ascontiguousarray(cc["ghost_owner"], np.int32)).to(dev)
        out_ = (torch.empty(1, dtype=torch.float64, device=dev), torch.empty((NN, 3), dtype=torch.float64, device=dev),
                torch.empty(6, dtype=torch.float64, device=dev))
        step_v = torch.tensor([drift_A * 0.6, drift_A * 0.64, drift_A * 0.48], dtype=torch.float64, device=dev)   # |v| = drift_A
        # (stream is torch's current stream: the position update and the evaluation are ordered on it)
        for _ in range(n_equil):
            p_ += step_v
            mm.compute(p_, t_, cc["box"], cc["n_local"], cc["n_ghost"], o_, out=out_, stream=stream)
        torch.cuda.synchronize(dev)
        s0 = mm.stats()
        a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a0.record(stream)
        for _ in range(n_prod):
            p_ += step_v
            mm.compute(p_, t_, cc["box"], cc["n_local"], cc["n_ghost"], o_, out=out_, stream=stream)
        a1.record(stream)
        torch.cuda.synchronize(dev)
        s1 = mm.stats()
        ms = a0.elapsed_time(a1) / n_prod
        return dict(n_local=cc["n_local"], equilibration_steps=n_equil, production_steps=n_prod, skin_A=skin_mA / 1000.0,
                    drift_A_per_step=drift_A, ms_per_step=ms, atom_steps_per_s=cc["n_local"] / (ms * 1e-3),
                    list_rebuilds=s1["n_list_rebuilds"] - s0["n_list_rebuilds"], list_reuses=s1["n_list_reuses"] - s0["n_list_reuses"],
                    graph_replays=s1["n_graph_replays"] - s0["n_graph_replays"])

    extra = {}
    if rank == 0 and world == 1 and not args.no_extra:
        ms_r, st_r = _time_mode(m, c, 1000, args.steps, max(args.warmup, 3))
        extra["list_reuse"] = dict(skin_A=1.0, ms_per_step=ms_r, value=n_local / (ms_r * 1e-3), unit=UNIT,
                                   graph_replays=st_r["n_graph_replays"], launches_per_step=st_r["n_launches"],
                                   note="static positions: every timed step re-filters the kept list at rc and replays the "
                                        "captured CUDA graph (no cell binning / sort / 27-cell scan, no host read)")
        m.set_option("skin_mA", 0)
        small = {}
        for kk in (1, 2, 3):
            if kk == k:
                continue
            cc, bb = _cached_workload(kk)
            mk = cc["model"]
            with P.Model(bb, mk["n_species"], mk["rc"], len(cc["pos"])) as mm:
                ms0, st0 = _time_mode(mm, cc, 0, 20, 5)
                ms1, st1 = _time_mode(mm, cc, 1000, 20, 5)
                mm.set_option("prune", 0); ms2, _ = _time_mode(mm, cc, 0, 20, 5) if cc["n_ghost"] else (None, None)
            small[f"config{kk}"] = dict(n_local=cc["n_local"], n_ghost=cc["n_ghost"], n_edges=st0["n_edges"],
                                        ms_rebuild_every_step=ms0, ms_list_reuse_graph=ms1,
                                        atom_steps_per_s_rebuild=cc["n_local"] / (ms0 * 1e-3),
                                        atom_steps_per_s_reuse=cc["n_local"] / (ms1 * 1e-3),
                                        launches_rebuild=st0["n_launches"], atoms_kept_by_pruning=st0["n_reached"],
                                        **({"ms_rebuild_unpruned": ms2} if ms2 is not None else {}))
        extra["other_configs"] = small
        # MD timing protocol of the paper (100 + 250 steps; at 1M atoms 10 + 40 to keep the default run short)
        md = {}
        for kk, (ne, npd) in ((1, (100, 250)), (2, (100, 250)), (k, (10, 40))):
            cc, bb = (c, blob) if kk == k else _cached_workload(kk)
            mk = cc["model"]
            if kk == k:
                md[f"config{kk}"] = _md_protocol(m, cc, ne, npd, 1000, 0.03)
                m.set_option("skin_mA", 0)
            else:
                with P.Model(bb, mk["n_species"], mk["rc"], len(cc["pos"])) as mm:
                    md[f"config{kk}"] = _md_protocol(mm, cc, ne, npd, 1000, 0.03)
        extra["md_protocol"] = md

    if rank == 0:
        cpu = None
        if world == 1 and not args.no_cpu_baseline:
            try:
                cpu, _ = _oracle_time(k, 3, 0)
            except Exception as ex:      # never lose the GPU measurement to the CPU leg
                cpu = dict(value=None, unit=UNIT, cores=os.cpu_count(), kind="oracle", sample=f"failed: {ex!r}")
        line = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=args.steps, warmup=max(args.warmup, 3),
                    ms_per_step=ms_step, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f32",
                    data="synthetic",
                    config=dict(workload=f"config {k}: {c['name']}, {n_local} local + {c['n_ghost']} ghost atoms, "
                                         f"{stats['n_edges']} directed edges, PaiNN {model['T']}x{model['F']} K={model['K']} rc={model['rc']}",
                                l2="working set (tens of GB) far larger than the 126 MB L2; no explicit flush",
                                multi_gpu="replicas only (one evaluation does not shard; BASELINE.json fixes 1 GPU)",
                                options="skin_mA=0 (list rebuilt in every step, as the metric demands)" + ("," + opts if opts else ""),
                                precision="fp64 cutoff predicate, fp32 edge math and node state, forward GEMMs exact (fp16 integer slices on tcgen05), adjoint GEMMs 3xTF32"),
                    clocks=clocks, e2e=e2e, gpu_launches=launches, roofline=roofline, cpu_baseline=cpu, **extra)
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
