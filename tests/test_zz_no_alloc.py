"""-m gpu: mlip_scan_i32_noalloc (include/mlip.h) -- the exclusive int32 prefix sum with its scratch in a fixed device
array instead of an allocation -- against the existing allocating path mlip_scan_i32, bit for bit (integer work), on
calls in a row that leave stale scratch behind. Collected last on purpose (file name): the suite runs with pytest -x."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

# ragged tails around the 2048-element tile, one and several tiles of tile totals, the 47,189,556 edges of BASELINE config 4
SIZES = [0, 1, 31, 2047, 2048, 2049, 65536 + 5, 1_000_003, 47_189_556]


def _values(torch, n, seed):
    g = torch.Generator(device="cuda").manual_seed(seed)
    return torch.randint(0, 61, (n,), dtype=torch.int32, device="cuda", generator=g)   # degrees of a radius graph


def test_noalloc_scan_equals_existing_path_on_calls_in_a_row():
    import torch
    import paper_2509_21694_b200 as mlip
    ctx = mlip.Context(0)
    # big first, then small ones: every later call finds the tile totals of an earlier, longer one in the scratch array
    for k, n in enumerate(sorted(SIZES, reverse=True) + SIZES):
        v = _values(torch, n, 1000 + k)
        ref = mlip.scan_i32(ctx, v)                      # existing path (scratch from the allocator)
        out = torch.full((n + 1,), -7, dtype=torch.int32, device="cuda")
        got = mlip.scan_i32_noalloc(ctx, v, out)
        again = mlip.scan_i32_noalloc(ctx, v)            # second call in a row on the same input
        ctx.status()
        assert torch.equal(got, ref) and torch.equal(again, ref), n
        # and against the definition, computed independently of both paths
        want = torch.zeros(n + 1, dtype=torch.int64, device="cuda")
        want[1:] = torch.cumsum(v.to(torch.int64), 0)
        assert torch.equal(got.to(torch.int64), want), n


def test_noalloc_scan_allocates_nothing_and_rejects_sizes_beyond_its_scratch():
    import torch
    import paper_2509_21694_b200 as mlip
    ctx = mlip.Context(0)
    n = 5_000_000
    v = _values(torch, n, 7)
    out = torch.empty(n + 1, dtype=torch.int32, device="cuda")
    mlip.scan_i32_noalloc(ctx, v, out)                   # first call: module load, address of the scratch array
    ctx.status()
    free0 = torch.cuda.mem_get_info(0)[0]
    for _ in range(3):
        mlip.scan_i32_noalloc(ctx, v, out)
    free1 = torch.cuda.mem_get_info(0)[0]                # before the stream is drained: a cudaMalloc would show here
    ctx.status()
    assert free1 == free0 == torch.cuda.mem_get_info(0)[0]
    assert int(out[n].item()) == int(v.sum().item())

    big = mlip.MLIP_SCAN_NOALLOC_MAX + 1
    vb = torch.zeros(big, dtype=torch.int32, device="cuda")
    ob = torch.full((big + 1,), -7, dtype=torch.int32, device="cuda")
    with pytest.raises(mlip.MlipError) as ei:
        mlip.scan_i32_noalloc(ctx, vb, ob)
    assert ei.value.code == -1 and "MLIP_SCAN_NOALLOC_MAX" in str(ei.value)
    ctx.status()
    assert int(ob[0].item()) == -7 and int(ob[big].item()) == -7      # nothing was launched
    at_max = mlip.scan_i32_noalloc(ctx, vb[:-1] + 1)                  # the limit itself is accepted
    ctx.status()
    assert int(at_max[-1].item()) == mlip.MLIP_SCAN_NOALLOC_MAX
    assert np.array_equal(at_max[:3].cpu().numpy(), [0, 1, 2])
