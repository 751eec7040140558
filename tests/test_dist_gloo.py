"""world_size-2 gloo test (CPU) of the N-GPU form of the path: sub-domains are dealt to the ranks
by k mod world, every rank computes the PARTIAL energy and forces of its sub-domains, one all-reduce (the product's
paper_2509_21694_b200.dist helper, the call bench.py makes under torchrun) sums them. The per-rank arithmetic is the
oracle's here (no GPU in this test); the sharding rule and the exchange are the product's."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import mlip_oracle as O
from synth_inputs import ModelSpec, make_weights, small_system


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_path):
    from paper_2509_21694_b200.dist import all_reduce_results, subdomains_of
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        spec = ModelSpec(4, 16, 8, 2, 3.0, 1.0 / np.sqrt(12.0))
        blob = make_weights(spec, 45)
        m = O.parse_weights(spec.n_species, spec.d, spec.n_rbf, spec.L_max, spec.r_cut, spec.agg_scale, blob)
        s = small_system(6, 0.08, seed=71)
        g = O.neighbor_list(s.pos, s.cell, spec.r_cut)
        parts = [(o, e) for o, e, _ in O.partition_grid_khop(s.pos, s.cell, (3, 1, 1), 6.0, spec.r_cut, g)]
        mine = subdomains_of(rank, world, len(parts))
        E, _, F, _ = O.energy_forces_partitioned(m, 2, s.pos, s.cell, s.species, [parts[k] for k in mine], g)
        sig = O.stress_partitioned(m, 2, s.pos, s.cell, s.species, [parts[k] for k in mine], g)
        tE = torch.tensor([E], dtype=torch.float64)
        tF = torch.tensor(F, dtype=torch.float32)
        tS = torch.tensor(sig, dtype=torch.float64)
        all_reduce_results(tE, tF, tS)
        if rank == 0:
            E0, _, F0, S0 = O.energy_forces_stress(m, 2, s.pos, s.cell, s.species, g)
            ok = (abs(tE.item() - E0) < 1e-10 * abs(E0) and np.abs(tF.numpy() - F0).max() < 1e-5 * np.sqrt(np.mean(F0 ** 2))
                  and np.abs(tS.numpy() - S0).max() < 1e-10 * np.abs(S0).max() and len(mine) == 2)
            open(out_path, "w").write("ok" if ok else f"bad {tE.item()} {E0}")
    finally:
        dist.destroy_process_group()


def test_two_rank_sharded_assembly_gloo(tmp_path):
    out = str(tmp_path / "result.txt")
    mp.spawn(_worker, args=(2, _free_port(), out), nprocs=2, join=True)
    assert open(out).read() == "ok"


def test_subdomain_dealing_rule():
    from paper_2509_21694_b200.dist import subdomains_of
    assert subdomains_of(0, 2, 8) == [0, 2, 4, 6] and subdomains_of(1, 2, 8) == [1, 3, 5, 7]
    assert sorted(sum((subdomains_of(r, 3, 8) for r in range(3)), [])) == list(range(8))
    assert subdomains_of(0, 1, 5) == list(range(5))
