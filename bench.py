"""bench.py -- atom-steps/s of the energy-and-force hot path (BASELINE.json `metric`).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--precision auto|fp32|bf16]
    python bench.py --impl reference ...        # the float64 oracle on the host cores

A step is one pass of the whole hot path over one synthetic
configuration: mlip_build_graph -> mlip_partition_grid -> mlip_energy_forces. `value` is timed
with positions/species already resident in HBM; `e2e` times mlip_step_host, i.e. the same pass
from pinned HOST buffers with the H2D copy of positions/species and the D2H copy of E and F
inside the timed region. One JSON line is printed by rank 0.

N > 1 (torchrun): the sub-domains are independent, so rank r evaluates the
sub-domains k with k mod N == r and one NCCL all-reduce sums E and F ("strong" scaling: the box is
fixed). Nothing in this build run has more than one GPU; the path is covered by the gloo test.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "atom-steps/s (E+F)"
UNIT = "atom-steps/s"
FALLBACK_PEAKS = {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}
# fp32 CUDA-core peak: 148 SMs x 128 FMA lanes x 2 flop x 1.965 GHz (B200_PROFILING.md unit counts / clocks)
ALU_FP32_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json config number (1-4); 4 = 1,048,576 atoms")
    ap.add_argument("--precision", default="auto", choices=["auto", "fp32", "bf16"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-active-sets", action="store_true",
                    help="evaluate every layer on the whole extended sub-graph (A/B against the per-layer active sets)")
    ap.add_argument("--n-cells", type=int, default=None, help="shrink the fcc box (debugging only; not a bench line)")
    return ap.parse_args()


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        p["_source"] = "measured"
        return p
    p = dict(FALLBACK_PEAKS)
    p["_source"] = "fallback"
    return p


def workload_name(cfg, n_atoms):
    g = "x".join(str(x) for x in cfg.grid)
    return (f"config{cfg.number}: {n_atoms} atoms {cfg.system.name}, L={cfg.L}, d={cfg.model.d}, "
            f"n_rbf={cfg.model.n_rbf}, r_cut={cfg.model.r_cut}, grid={g}, halo={cfg.halo}")


# ------------------------------------------------------------------------------------------
# oracle legs (the only place bench.py touches oracle/)
# ------------------------------------------------------------------------------------------
def oracle_sample(cfg_number: int, n_cells: int):
    """Time the float64 oracle, as it stands, on a bounded sample of the workload: the same recipe
    with a smaller fcc box, unpartitioned. Returns (atom-steps/s, n_atoms, seconds, cores)."""
    from oracle import mlip_oracle as O
    from synth_inputs import make_config
    cfg = make_config(cfg_number, n_cells_override=n_cells)
    s, m = cfg.system, cfg.model
    om = O.parse_weights(m.n_species, m.d, m.n_rbf, m.L_max, m.r_cut, m.agg_scale, cfg.weights)
    t0 = time.perf_counter()
    O.energy_forces(om, cfg.L, s.pos, s.cell, s.species)
    dt = time.perf_counter() - t0
    return len(s.pos) / dt, len(s.pos), dt, len(os.sched_getaffinity(0))


def sample_cells(cfg_number: int) -> int:
    return {1: 3, 2: 5, 3: 4, 4: 6}.get(cfg_number, 4)


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from synth_inputs import make_config
    nc = sample_cells(args.config)
    cfg_full = make_config(args.config, with_weights=False, n_cells_override=args.n_cells)
    vals = []
    n_atoms = 0
    cores = 0
    for i in range(args.warmup + args.steps):
        v, n_atoms, dt, cores = oracle_sample(args.config, nc)
        if i >= args.warmup:
            vals.append((v, dt))
    value = float(np.mean([v for v, _ in vals]))
    sample = f"same recipe at fcc {nc}^3 ({n_atoms} atoms), unpartitioned, float64 NumPy oracle, one evaluation per step"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": float(np.mean([dt for _, dt in vals]) * 1e3), "higher_is_better": True,
        "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(cfg_full, len(cfg_full.system.pos)), "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------
# clocks sampling during the timed region
# ------------------------------------------------------------------------------------------
class ClockSampler:
    def __init__(self, device: int):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thread = None
        self.device = device
        try:
            import pynvml
            pynvml.nvmlInit()
            # honour CUDA_VISIBLE_DEVICES when it is a plain index list
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            idx = device
            if vis:
                try:
                    idx = int(vis.split(",")[device])
                except Exception:
                    idx = device
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(idx)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def _loop(self):
        nv = self.nv
        names = {}
        for k in dir(nv):
            if k.startswith("nvmlClocksThrottleReason") or k.startswith("nvmlClocksEventReason"):
                v = getattr(nv, k)
                if isinstance(v, int) and v:
                    names.setdefault(v, k.replace("nvmlClocksThrottleReason", "").replace("nvmlClocksEventReason", ""))
        while not self._stop.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    mask = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if mask & bit and name not in ("None", "All"):
                        self.reasons.add(name)
            except Exception:
                pass
            self._stop.wait(0.05)

    def start(self):
        if self.nv is not None:
            self._thread = threading.Thread(target=self._loop, daemon=True)
            self._thread.start()

    def stop(self):
        self._stop.set()
        if self._thread is not None:
            self._thread.join()
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ------------------------------------------------------------------------------------------
# the CUDA path
# ------------------------------------------------------------------------------------------
def ncu_traffic(config: int, group: str):
    """DRAM bytes per launch of a kernel group from the committed ncu --set full capture (profiles/*_traffic.csv,
    newest round last), or None when no capture of this config exists."""
    import csv
    import glob
    best = None
    for path in sorted(glob.glob(os.path.join(ROOT, "profiles", "*_traffic.csv"))):
        for row in csv.DictReader(open(path)):
            if int(row["config"]) == config and row["kernel_group"] == group:
                best = float(row["dram_bytes_per_launch"])
    return best


def flops_edge_layer(d: int, n_rbf: int) -> float:
    """Algorithmic flop per edge per layer of one direction: the first edge
    linear factorises into per-node projections, so only the n_rbf x d term and the d x d second
    linear are per-edge work."""
    return 2.0 * d * n_rbf + 2.0 * d * d


def run_ours(args):
    import torch
    import torch.distributed as dist

    import paper_2509_21694_b200 as mlip
    from paper_2509_21694_b200.dist import all_reduce_results
    from synth_inputs import make_config

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the hot path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = f"cuda:{local_rank}"
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(dev))
    assert world == args.gpus or world == 1, "launch with torchrun --nproc-per-node N for --gpus N"

    cfg = make_config(args.config, n_cells_override=args.n_cells)
    s, m = cfg.system, cfg.model
    prec_name = cfg.precision if args.precision == "auto" else args.precision
    prec = mlip.MLIP_BF16 if prec_name == "bf16" else mlip.MLIP_FP32
    N = len(s.pos)
    partitioned = tuple(cfg.grid) != (1, 1, 1)
    if world > 1 and not partitioned:
        raise SystemExit("bench.py: --gpus > 1 needs a partitioned config (sub-domains are the unit that shards)")

    ctx = mlip.Context(local_rank)
    ctx.set_active_sets(not args.no_active_sets)
    model = mlip.Model(ctx, m.n_species, m.d, m.n_rbf, m.L_max, m.r_cut, m.agg_scale, cfg.weights)
    pos = torch.tensor(s.pos, dtype=torch.float64, device=dev)
    species = torch.tensor(s.species, dtype=torch.int32, device=dev)
    out = (torch.empty(1, dtype=torch.float64, device=dev), torch.empty((N, 3), dtype=torch.float32, device=dev), None)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)  # 256 MiB > 126 MB L2
    info = {}

    def step():
        g = mlip.Graph(ctx, pos, s.cell, species, m.r_cut)
        part = mlip.Partition(ctx, g, cfg.halo, grid=cfg.grid) if partitioned else None
        if world > 1:
            E, F, _ = mlip.energy_forces_shard(ctx, model, cfg.L, g, part, rank, world, prec, out=out)
            all_reduce_results(E, F)
        else:
            E, F, _ = mlip.energy_forces(ctx, model, cfg.L, g, part, prec, want_atom_energy=False, out=out)
        info["edges"] = g.num_edges
        info["subs"] = part.info() if part is not None else [dict(n_owned=N, n_ext=N, n_edges=g.num_edges)]
        # edge evaluations per layer and sub-domain (per-layer active sets: mlip_part_layer_info)
        info["layers"] = (part.layer_info(cfg.L) if part is not None
                          else [[dict(n_recv=N, n_send=N, n_edges=g.num_edges)] * cfg.L])
        return E, F

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
        flush.zero_()
    barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    ctx.profile(True)
    launches0 = ctx.launches
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    for a, b in ev:
        flush.zero_()  # evict L2 between timed iterations (outside the event pair)
        a.record()
        E, F = step()
        b.record()
    barrier()
    launches = ctx.launches - launches0
    groups = ctx.profile_read()
    ctx.profile(False)
    clocks = sampler.stop()
    ms = torch.tensor([sum(a.elapsed_time(b) for a, b in ev) / args.steps], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(ms, op=dist.ReduceOp.MAX)
    ms_per_step = float(ms.item())
    value = N / (ms_per_step * 1e-3)
    E_val = float(E.item())
    F_sum = F.sum(0).cpu().numpy().tolist()

    # ---- end to end through mlip_step_host with pinned host buffers ----
    e2e = None
    if not args.no_e2e and world == 1:
        pos_h = torch.from_numpy(s.pos.copy()).pin_memory()
        sp_h = torch.from_numpy(s.species.copy()).pin_memory()
        F_h = torch.empty((N, 3), dtype=torch.float32).pin_memory()
        t_list = []
        for i in range(1 + max(1, min(args.steps, 3))):
            flush.zero_()
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            mlip.step_host(ctx, model, cfg.L, pos_h.numpy(), s.cell, sp_h.numpy(), grid=cfg.grid, halo=cfg.halo,
                           precision=prec, forces_out=F_h.numpy())
            t_list.append(time.perf_counter() - t0)  # step_host synchronises before returning
        t_e2e = float(np.mean(t_list[1:]))
        e2e = {"value": N / t_e2e, "unit": UNIT, "h2d_bytes_per_step": int(pos_h.numel() * 8 + sp_h.numel() * 4),
               "d2h_bytes_per_step": int(F_h.numel() * 4 + 8), "ms_per_step": t_e2e * 1e3}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel group ----
    pk = peaks()
    edges_total = sum(x["n_edges"] for x in info["subs"][rank::world]) if world > 1 else sum(x["n_edges"] for x in info["subs"])
    mine = info["layers"][rank::world] if world > 1 else info["layers"]
    edge_layers = sum(r["n_edges"] for rows in mine for r in rows)   # edge-layer evaluations actually launched
    per_step = {k: v[0] / args.steps for k, v in groups.items()}
    dom = max(("edge_fwd", "edge_bwd"), key=lambda k: per_step[k])
    flop = edge_layers * flops_edge_layer(m.d, m.n_rbf)
    achieved = flop / (per_step[dom] * 1e-3) / 1e12 if per_step[dom] > 0 else 0.0
    if prec_name == "bf16":
        bound, peak, peak_src = "tensor", pk["bf16_tflops_sustained"], pk["_source"] + " (sustained cuBLAS bf16)"
    else:
        bound, peak, peak_src = "alu", ALU_FP32_TFLOPS, "derived: 148 SM x 128 FMA x 2 x 1.965 GHz"
    roofline = {"kernel": dom, "bound": bound, "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                "frac": achieved / peak, "traffic": ncu_traffic(args.config, dom), "traffic_unit": "dram bytes per launch (ncu)",
                "peak_source": peak_src,
                "algorithmic_flop_per_step": flop, "kernel_ms_per_step": per_step[dom],
                "executed_over_algorithmic": 2.0 if dom == "edge_bwd" else 1.0}

    cpu = None
    if not args.no_cpu_baseline and world == 1:
        nc = sample_cells(args.config)
        v, n_s, dt, cores = oracle_sample(args.config, nc)
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"same recipe at fcc {nc}^3 ({n_s} atoms), unpartitioned, one evaluation ({dt:.1f} s)"}

    n_own = [x["n_owned"] for x in info["subs"]]
    n_ext = [x["n_ext"] for x in info["subs"]]
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
        "dtype": "bf16" if prec_name == "bf16" else "f32", "data": "synthetic",
        "config": {"workload": workload_name(cfg, N), "n_atoms": N, "n_edges": info["edges"],
                   "sub_domains": len(info["subs"]), "edges_in_subgraphs": int(edges_total),
                   "edge_layers_evaluated_per_step": int(edge_layers), "active_sets": not args.no_active_sets,
                   "halo_growth_H": float(np.mean([(e - o) / max(o, 1) for o, e in zip(n_own, n_ext)])),
                   "l2": "256 MiB buffer rewritten between timed iterations; working set also exceeds the 126 MB L2"
                   if N > 200000 else "256 MiB buffer rewritten between timed iterations",
                   "step": "mlip_build_graph + mlip_partition_grid + mlip_energy_forces, inputs resident in HBM"},
        "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline, "cpu_baseline": cpu,
        "kernel_ms_per_step": per_step, "energy": E_val, "force_sum": F_sum,
    }
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
