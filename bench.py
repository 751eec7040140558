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


def dtype_label(prec_name: str, d: int) -> str:
    if prec_name == "bf16":
        return "f16 operands, f32 accumulate (MLIP_BF16)"
    if d == 128:
        return "f32 (MLIP_FP32; edge contractions as 3-term bf16 splits on tcgen05 with f32 accumulate)"
    return "f32"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json config number (1-5); 4 = 1,048,576 atoms (the metric's), 5 = three-body variant")
    ap.add_argument("--precision", default="auto", choices=["auto", "fp32", "bf16"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-active-sets", action="store_true",
                    help="evaluate every layer on the whole extended sub-graph (A/B against the per-layer active sets)")
    ap.add_argument("--md", action="store_true",
                    help="time the on-device MD driver mlip_md_run (Langevin, --steps steps) instead of single evaluations; "
                         "--skin / --cuda-graph select Verlet-skin reuse and CUDA-graph replay")
    ap.add_argument("--skin", type=float, default=0.0)
    ap.add_argument("--cuda-graph", action="store_true")
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
    om = O.parse_weights(m.n_species, m.d, m.n_rbf, m.L_max, m.r_cut, m.agg_scale, cfg.weights, r_cut3=m.r_cut3)
    graph = O.neighbor_list(s.pos, s.cell, m.r_cut)
    t0 = time.perf_counter()
    O.energy_forces(om, cfg.L, s.pos, s.cell, s.species)
    dt = time.perf_counter() - t0
    return len(s.pos) / dt, len(s.pos), dt, len(os.sched_getaffinity(0)), len(graph[0]) * cfg.L / dt


def sample_cells(cfg_number: int, n_evaluations: int = 1) -> int:
    """fcc cells per axis of the oracle's bounded sample: 10-30 s of host time per evaluation on ~16 cores when it is
    evaluated once (the cpu_baseline leg) or a handful of times, about 4 s each when `--impl reference` repeats it
    for many steps (the whole run has to end within a few minutes)."""
    if n_evaluations > 8:
        return {1: 3, 2: 5, 3: 4, 4: 6, 5: 5}.get(cfg_number, 4)
    return {1: 3, 2: 8, 3: 6, 4: 12, 5: 9}.get(cfg_number, 4)


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from synth_inputs import make_config
    nc = sample_cells(args.config, args.warmup + args.steps)
    cfg_full = make_config(args.config, with_weights=False, n_cells_override=args.n_cells)
    vals = []
    n_atoms = 0
    cores = 0
    for i in range(args.warmup + args.steps):
        v, n_atoms, dt, cores, _ = oracle_sample(args.config, nc)
        if i >= args.warmup:
            vals.append((v, dt))
    value = float(np.mean([v for v, _ in vals]))
    sample = f"same recipe at {nc}^3 cells ({n_atoms} atoms), unpartitioned, float64 NumPy oracle, one evaluation per step"
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
    """(DRAM bytes per launch, capture label) of a kernel group from the committed ncu --set full captures
    (profiles/*_traffic.csv, newest round last; the label names the commit the capture was made on), or (None, None)
    when no capture of this config exists."""
    import csv
    import glob
    best, label = None, None
    for path in sorted(glob.glob(os.path.join(ROOT, "profiles", "*_traffic.csv"))):
        for row in csv.DictReader(open(path)):
            if int(row["config"]) == config and row["kernel_group"] == group:
                best = float(row["dram_bytes_per_launch"])
                label = f"{os.path.basename(path)} @ {row.get('commit') or 'commit not recorded'}"
    return best, label


MUFU_PER_SM_PER_CLK = 16   # MUFU (tanh/ex2) results per clock and SM: 4 per SM sub-partition (B300_MICROARCH.md pipes)


def edge_rooflines(name, ms, edge_layers, launches, d, n_rbf, pk, sm_mhz, spill_layers=0):
    """The three rooflines SURVEY.md 8(d) asks for on the fused edge kernels (they sit at the ridge): tensor pipe, MUFU
    and HBM, each as algorithmic work / measured time / peak.
      tensor  2 d n_rbf + 2 d^2 flop per edge-layer and direction (the reverse pass EXECUTES twice that: recompute)
      MUFU    2 d transcendental results per edge-layer and direction (one tanh per SiLU; reverse pass: the recomputed ones)
      HBM     sender row 2 d B + 28 B metadata per edge-layer; reverse pass adds the 2 d B abar spill of the layers with a
              node adjoint and 4 B of rbar"""
    if ms <= 0:
        return []
    t = ms * 1e-3
    flop = edge_layers * flops_edge_layer(d, n_rbf)
    mufu = edge_layers * 2.0 * d
    hbm = edge_layers * (2.0 * d + 28.0) + spill_layers * 2.0 * d + (4.0 * edge_layers if name == "edge_bwd" else 0.0)
    mufu_peak = 148 * MUFU_PER_SM_PER_CLK * sm_mhz * 1e6
    return [
        {"kernel": name, "bound": "tensor", "achieved": flop / t / 1e12, "peak": pk["bf16_tflops_sustained"], "unit": "TFLOP/s",
         "frac": flop / t / 1e12 / pk["bf16_tflops_sustained"], "launches_per_step": launches},
        {"kernel": name, "bound": "mufu", "achieved": mufu / t / 1e12, "peak": mufu_peak / 1e12, "unit": "Tresult/s",
         "frac": mufu / t / mufu_peak, "peak_source": f"derived: 148 SM x 16 /clk x {sm_mhz:.0f} MHz (median SM clock of the run)"},
        {"kernel": name, "bound": "hbm", "achieved": hbm / t / 1e9, "peak": pk["hbm_gbs"], "unit": "GB/s",
         "frac": hbm / t / 1e9 / pk["hbm_gbs"]},
    ]


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
    model = mlip.Model(ctx, m.n_species, m.d, m.n_rbf, m.L_max, m.r_cut, m.agg_scale, cfg.weights, r_cut3=m.r_cut3)
    pos = torch.tensor(s.pos, dtype=torch.float64, device=dev)
    species = torch.tensor(s.species, dtype=torch.int32, device=dev)
    out = (torch.empty(1, dtype=torch.float64, device=dev), torch.empty((N, 3), dtype=torch.float32, device=dev), None)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)  # 256 MiB > 126 MB L2
    info = {}

    def step(collect=False):
        g = mlip.Graph(ctx, pos, s.cell, species, m.r_cut)
        # N > 1: every rank builds its own sub-domains only (mlip_partition_grid_shard)
        part = mlip.Partition(ctx, g, cfg.halo, grid=cfg.grid, shard=rank, n_shards=world) if partitioned else None
        if world > 1:
            E, F, _ = mlip.energy_forces_shard(ctx, model, cfg.L, g, part, rank, world, prec, out=out)
            all_reduce_results(E, F)
        else:
            E, F, _ = mlip.energy_forces(ctx, model, cfg.L, g, part, prec, want_atom_energy=False, out=out)
        if collect:   # sizes for the roofline arithmetic: only in the separate profiling pass, never in the timed region
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
    launches0 = ctx.launches
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    for a, b in ev:
        flush.zero_()  # evict L2 between timed iterations (outside the event pair)
        a.record()
        E, F = step()
        b.record()
    barrier()
    launches = ctx.launches - launches0
    clocks = sampler.stop()
    # separate pass with the per-kernel-group event timers on (they cost a few event records per launch group, so they
    # stay out of the timed region above): kernel_ms_per_step and the roofline numerators come from here
    prof_steps = max(1, min(args.steps, 3))
    ctx.profile(True)
    for _ in range(prof_steps):
        flush.zero_()
        step(collect=True)
    barrier()
    groups = ctx.profile_read()
    ctx.profile(False)
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
    per_step = {k: v[0] / prof_steps for k, v in groups.items()}
    n_launch = {k: v[1] / prof_steps for k, v in groups.items()}
    dom = max(("edge_fwd", "edge_bwd"), key=lambda k: per_step[k])
    flop = edge_layers * flops_edge_layer(m.d, m.n_rbf)
    achieved = flop / (per_step[dom] * 1e-3) / 1e12 if per_step[dom] > 0 else 0.0
    if prec_name == "bf16":
        bound, peak, peak_src = "tensor", pk["bf16_tflops_sustained"], pk["_source"] + " (sustained cuBLAS bf16)"
    elif m.d == 128:
        # MLIP_FP32 at d = 128 runs its contractions on tcgen05 with every fp32 operand split into three bf16 terms
        # (edge_x3.cu): six bf16 MMAs per fp32 product, so the fp32-equivalent tensor peak is the bf16 peak / 6
        bound, peak = "tensor", pk["bf16_tflops_sustained"] / 6.0
        peak_src = pk["_source"] + " (sustained cuBLAS bf16) / 6: six bf16 MMAs per fp32 product (3-term operand split)"
    else:
        bound, peak, peak_src = "alu", ALU_FP32_TFLOPS, "derived: 148 SM x 128 FMA x 2 x 1.965 GHz"
    traffic, traffic_capture = ncu_traffic(args.config, dom)
    roofline = {"kernel": dom, "bound": bound, "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                "frac": achieved / peak, "traffic": traffic, "traffic_unit": "dram bytes per launch (ncu)",
                "traffic_capture": traffic_capture, "peak_source": peak_src,
                "algorithmic_flop_per_step": flop, "kernel_ms_per_step": per_step[dom],
                "executed_over_algorithmic": 2.0 if dom == "edge_bwd" else 1.0}
    # every binding unit of the big kernel groups (SURVEY.md 8(d) "report all three" for the fused edge kernels)
    rooflines = []
    if prec_name == "bf16":
        sm_mhz = clocks.get("sm_mhz") or pk.get("sm_max_mhz", 1965.0)
        # layers with a node adjoint (all but the first) spill abar and are read back by the sender-side gather
        spill_layers = sum(r["n_edges"] for rows in mine for r in rows[1:])
        rooflines += edge_rooflines("edge_fwd", per_step["edge_fwd"], edge_layers, n_launch["edge_fwd"], m.d, m.n_rbf, pk, sm_mhz)
        rooflines += edge_rooflines("edge_bwd", per_step["edge_bwd"], edge_layers, n_launch["edge_bwd"], m.d, m.n_rbf, pk, sm_mhz,
                                    spill_layers)
        if per_step["gather_rev"] > 0:
            send_rows = sum(r["n_send"] for rows in mine for r in rows[1:])
            gb = (spill_layers * (2.0 * m.d + 4.0) + send_rows * 2.0 * m.d) / 1e9
            rooflines.append({"kernel": "gather_rev", "bound": "hbm", "achieved": gb / (per_step["gather_rev"] * 1e-3),
                              "peak": pk["hbm_gbs"], "unit": "GB/s", "frac": gb / (per_step["gather_rev"] * 1e-3) / pk["hbm_gbs"]})
        if per_step["node_gemm"] > 0:
            # 10 d^2 flop per atom-layer forward (P, Q, V1, V2) and the same again in the reverse pass, + readout 2 d^2 x 2
            atom_layers = sum(r["n_send"] for rows in mine for r in rows)
            nflop = atom_layers * 20.0 * m.d * m.d
            rooflines.append({"kernel": "node_gemm", "bound": "tensor", "achieved": nflop / (per_step["node_gemm"] * 1e-3) / 1e12,
                              "peak": pk["bf16_tflops_sustained"], "unit": "TFLOP/s",
                              "frac": nflop / (per_step["node_gemm"] * 1e-3) / 1e12 / pk["bf16_tflops_sustained"]})

    cpu = None
    if not args.no_cpu_baseline and world == 1:
        nc = sample_cells(args.config)
        v, n_s, dt, cores, el_rate = oracle_sample(args.config, nc)
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"same recipe at {nc}^3 cells ({n_s} atoms), unpartitioned, one evaluation ({dt:.1f} s)",
               "edge_layers_per_s": el_rate,
               # the partitioned workload evaluates edge_layers / N edge-layers per atom (halo included)
               "extrapolated_to_workload": el_rate * N / max(edge_layers, 1),
               "extrapolated_note": "sample edge-layers/s x N / edge-layers evaluated per step of this workload"}

    own_subs = info["subs"][rank::world] if world > 1 else info["subs"]   # N > 1: a rank builds its own sub-domains only
    n_own = [x["n_owned"] for x in own_subs]
    n_ext = [x["n_ext"] for x in own_subs]
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
        "dtype": dtype_label(prec_name, m.d), "data": "synthetic",
        "config": {"workload": workload_name(cfg, N), "n_atoms": N, "n_edges": info["edges"],
                   "sub_domains": len(info["subs"]), "edges_in_subgraphs": int(edges_total),
                   "edge_layers_evaluated_per_step": int(edge_layers), "active_sets": not args.no_active_sets,
                   "halo_growth_H": float(np.mean([(e - o) / max(o, 1) for o, e in zip(n_own, n_ext)])),
                   "l2": "256 MiB buffer rewritten between timed iterations; working set also exceeds the 126 MB L2"
                   if N > 200000 else "256 MiB buffer rewritten between timed iterations",
                   "step": "mlip_build_graph + mlip_partition_grid + mlip_energy_forces, inputs resident in HBM"},
        "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline, "rooflines": rooflines,
        "cpu_baseline": cpu,
        "kernel_ms_per_step": per_step, "energy": E_val, "force_sum": F_sum,
    }
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_md(args):
    """atom-steps/s of the MD driver: K Langevin steps of 2 fs at 300 K on the configuration's
    system, device-timed inside mlip_md_run (CUDA events around the K steps). Not the BASELINE metric: a secondary line."""
    import torch

    import paper_2509_21694_b200 as mlip
    from synth_inputs import make_config

    cfg = make_config(args.config, n_cells_override=args.n_cells)
    s, m = cfg.system, cfg.model
    prec_name = cfg.precision if args.precision == "auto" else args.precision
    prec = mlip.MLIP_BF16 if prec_name == "bf16" else mlip.MLIP_FP32
    N = len(s.pos)
    dev = "cuda:0"
    ctx = mlip.Context(0)
    model = mlip.Model(ctx, m.n_species, m.d, m.n_rbf, m.L_max, m.r_cut, m.agg_scale, cfg.weights, r_cut3=m.r_cut3)
    rng = np.random.default_rng(5000 + args.config)
    mass = torch.full((N,), 30.0, dtype=torch.float64, device=dev)
    species = torch.tensor(s.species, dtype=torch.int32, device=dev)
    kw = dict(grid=cfg.grid, halo=cfg.halo, precision=prec, thermostat=mlip.MLIP_MD_LANGEVIN, temperature=300.0, friction=0.01,
              seed=1, skin=args.skin, cuda_graph=args.cuda_graph)
    out = None
    for it in range(2):   # the first run warms up (allocator pool, kernel images)
        pos = torch.tensor(s.pos, dtype=torch.float64, device=dev).contiguous()
        vel = torch.tensor(rng.normal(0, 0.003, s.pos.shape), dtype=torch.float64, device=dev).contiguous()
        launches0 = ctx.launches
        e, st = mlip.md_run(ctx, model, cfg.L, pos, vel, mass, s.cell, species, 2.0, args.steps if it else max(2, args.warmup), **kw)
        out = (e, st, ctx.launches - launches0)
    e, st, launches = out
    ms = st["ms_total"] / args.steps
    line = {"metric": "atom-steps/s (MD, Langevin)", "value": N / (ms * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
            "dtype": dtype_label(prec_name, m.d), "data": "synthetic",
            "config": {"workload": workload_name(cfg, N), "dt_fs": 2.0, "temperature_K": 300.0, "skin": args.skin,
                       "cuda_graph": bool(args.cuda_graph)},
            "md_stats": st, "gpu_launches": int(launches), "energy_first_last": [float(e[0]), float(e[-1])]}
    print(json.dumps(line), flush=True)


def main():
    args = parse_args()
    if args.md:
        run_md(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
