"""ctypes binding of include/mlip.h. Same names as the C entry points; marshalling only.

PyTorch is used for device memory and the stream; no arithmetic of the method happens here.
There is no CPU fallback: if the shared library is missing or no sm_100 device is present the
calls raise MlipError.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

MLIP_FP32 = 0
MLIP_BF16 = 1
MLIP_MAGIC = 0x50494C4D
GROUPS = ("edge_fwd", "edge_bwd", "gather_rev", "node_gemm", "readout_forces", "graph", "partition", "three_body")

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = None


class MlipError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"mlip status {code}: {msg}")
        self.code = code


class mlip_model_header(C.Structure):
    _fields_ = [("magic", C.c_uint32), ("version", C.c_uint32), ("n_species", C.c_int32), ("d", C.c_int32),
                ("n_rbf", C.c_int32), ("L_max", C.c_int32), ("r_cut", C.c_float), ("agg_scale", C.c_float),
                ("flags", C.c_int32), ("n_rbf3", C.c_int32), ("l_max", C.c_int32), ("r_cut3", C.c_float)]


class mlip_md_params(C.Structure):
    _fields_ = [("dt", C.c_double), ("n_steps", C.c_int32), ("thermostat", C.c_int32), ("temperature", C.c_double),
                ("friction", C.c_double), ("seed", C.c_uint64), ("skin", C.c_double), ("cuda_graph", C.c_int32),
                ("reserved", C.c_int32)]


class mlip_md_stats(C.Structure):
    _fields_ = [("n_rebuilds", C.c_int64), ("n_graph_replays", C.c_int64), ("ms_total", C.c_double)]


MLIP_MD_NVE = 0
MLIP_MD_LANGEVIN = 1


def lib_path() -> str:
    """The in-tree library; MLIP_B200_LIB selects another build of the same sources (A/B measurements)."""
    return os.environ.get("MLIP_B200_LIB") or os.path.join(_HERE, "libmlip_b200.so")


def load_library():
    """dlopen the in-tree library and declare the prototypes of every symbol of include/mlip.h."""
    global _LIB
    if _LIB is not None:
        return _LIB
    path = lib_path()
    if not os.path.exists(path):
        raise MlipError(-6, f"{path} not built: run `python -m paper_2509_21694_b200.build` (no CPU fallback exists)")
    lib = C.CDLL(path)
    vp, i32, i64, dbl = C.c_void_p, C.c_int, C.c_int64, C.c_double
    P = C.POINTER
    lib.mlip_model_num_weights.restype = C.c_size_t
    lib.mlip_model_num_weights.argtypes = [P(mlip_model_header)]
    lib.mlip_ctx_create.argtypes = [i32, vp, P(vp)]
    lib.mlip_ctx_destroy.argtypes = [vp]; lib.mlip_ctx_destroy.restype = None
    lib.mlip_last_error.argtypes = [vp]; lib.mlip_last_error.restype = C.c_char_p
    lib.mlip_ctx_status.argtypes = [vp]
    lib.mlip_model_load.argtypes = [vp, P(mlip_model_header), vp, C.c_size_t, P(vp)]
    lib.mlip_model_destroy.argtypes = [vp]; lib.mlip_model_destroy.restype = None
    lib.mlip_build_graph.argtypes = [vp, vp, vp, vp, i64, dbl, P(vp)]
    lib.mlip_graph_num_edges.argtypes = [vp, P(i64)]
    lib.mlip_graph_export_edges.argtypes = [vp, vp, vp, vp, vp]
    lib.mlip_graph_destroy.argtypes = [vp]; lib.mlip_graph_destroy.restype = None
    lib.mlip_partition.argtypes = [vp, vp, i32, dbl, P(vp)]
    lib.mlip_partition_grid.argtypes = [vp, vp, P(i32), dbl, P(vp)]
    lib.mlip_partition_grid_shard.argtypes = [vp, vp, P(i32), dbl, i32, i32, P(vp)]
    lib.mlip_part_count.argtypes = [vp, P(i32)]
    lib.mlip_part_info.argtypes = [vp, i32, P(i64), P(i64), P(i64)]
    lib.mlip_part_layer_info.argtypes = [vp, i32, i32, i32, P(i64), P(i64), P(i64)]
    lib.mlip_part_destroy.argtypes = [vp]; lib.mlip_part_destroy.restype = None
    lib.mlip_ctx_set_active_sets.argtypes = [vp, i32]
    lib.mlip_ctx_set_khop_halo.argtypes = [vp, i32]
    lib.mlip_energy_forces.argtypes = [vp, vp, i32, vp, vp, i32, vp, vp, vp]
    lib.mlip_energy_forces_shard.argtypes = [vp, vp, i32, vp, vp, i32, i32, i32, vp, vp, vp]
    lib.mlip_energy_forces_stress.argtypes = [vp, vp, i32, vp, vp, i32, i32, i32, vp, vp, vp, vp]
    lib.mlip_md_nve.argtypes = [vp, vp, i32, vp, vp, vp, vp, vp, i64, P(i32), dbl, i32, dbl, i32, vp]
    lib.mlip_md_run.argtypes = [vp, vp, i32, vp, vp, vp, vp, vp, i64, P(i32), dbl, i32, P(mlip_md_params), vp, P(mlip_md_stats)]
    lib.mlip_step_host.argtypes = [vp, vp, i32, vp, vp, vp, i64, P(i32), dbl, i32, vp, vp]
    lib.mlip_ctx_launch_count.argtypes = [vp]; lib.mlip_ctx_launch_count.restype = i64
    lib.mlip_ctx_profile.argtypes = [vp, i32]
    lib.mlip_ctx_profile_read.argtypes = [vp, i32, P(dbl), P(i64)]
    lib.mlip_scan_i32.argtypes = [vp, vp, vp, i64]
    lib.mlip_scan_i32_noalloc.argtypes = [vp, vp, vp, i64]
    _LIB = lib
    return lib


def _torch():
    import torch
    return torch


class Context:
    """mlip_ctx bound to the current torch CUDA stream of `device`."""

    def __init__(self, device: int = 0, stream=None):
        self.lib = load_library()
        torch = _torch()
        if not torch.cuda.is_available():
            raise MlipError(-6, "no CUDA device: the hot path has no CPU fallback")
        self.device = device
        self.torch_stream = stream if stream is not None else torch.cuda.current_stream(device)
        h = C.c_void_p()
        st = self.lib.mlip_ctx_create(device, C.c_void_p(self.torch_stream.cuda_stream), C.byref(h))
        if st != 0:
            raise MlipError(st, "mlip_ctx_create failed (needs an sm_100 device)")
        self.h = h
        self._refs = 1  # the context itself + one per live child handle (GC may finalise in any order)

    def _retain(self):
        self._refs += 1

    def _release(self):
        self._refs -= 1
        if self._refs == 0 and self.h:
            self.lib.mlip_ctx_destroy(self.h)
            self.h = None

    def check(self, status):
        if status != 0:
            raise MlipError(status, self.lib.mlip_last_error(self.h).decode())

    def status(self):
        """mlip_ctx_status: synchronise the stream and raise if the asynchronous work reported an error."""
        self.check(self.lib.mlip_ctx_status(self.h))

    @property
    def launches(self) -> int:
        return int(self.lib.mlip_ctx_launch_count(self.h))

    def set_active_sets(self, enable: bool):
        """mlip_ctx_set_active_sets: per-layer active sets inside sub-domains (on by default)."""
        self.check(self.lib.mlip_ctx_set_active_sets(self.h, 1 if enable else 0))

    def set_khop_halo(self, enable: bool):
        """mlip_ctx_set_khop_halo: K-hop search (default) or whole geometric box for the next partitions."""
        self.check(self.lib.mlip_ctx_set_khop_halo(self.h, 1 if enable else 0))

    def profile(self, enable: bool):
        """mlip_ctx_profile: start (clearing the counters) or stop per-kernel-group event timing."""
        self.check(self.lib.mlip_ctx_profile(self.h, 1 if enable else 0))

    def profile_read(self) -> dict:
        """mlip_ctx_profile_read for every group -> {name: (ms_total, n_launches)}."""
        out = {}
        for gid, name in enumerate(GROUPS):
            ms, n = C.c_double(), C.c_int64()
            self.check(self.lib.mlip_ctx_profile_read(self.h, gid, C.byref(ms), C.byref(n)))
            out[name] = (ms.value, int(n.value))
        return out

    def __del__(self):
        if getattr(self, "_refs", 0) > 0:
            self._release()


def make_header(n_species, d, n_rbf, L_max, r_cut, agg_scale, r_cut3=0.0) -> mlip_model_header:
    """r_cut3 > 0 selects the three-body variant (flags bit 0, n_rbf3 = 4, l_max = 3)."""
    if r_cut3 > 0.0:
        return mlip_model_header(MLIP_MAGIC, 1, n_species, d, n_rbf, L_max, float(r_cut), float(agg_scale), 1, 4, 3, float(r_cut3))
    return mlip_model_header(MLIP_MAGIC, 1, n_species, d, n_rbf, L_max, float(r_cut), float(agg_scale), 0, 0, 0, 0.0)


class Model:
    def __init__(self, ctx: Context, n_species, d, n_rbf, L_max, r_cut, agg_scale, blob: np.ndarray, r_cut3: float = 0.0):
        self.ctx = ctx
        self.header = make_header(n_species, d, n_rbf, L_max, r_cut, agg_scale, r_cut3)
        blob = np.ascontiguousarray(blob, dtype=np.float32)
        h = C.c_void_p()
        ctx.check(ctx.lib.mlip_model_load(ctx.h, C.byref(self.header), blob.ctypes.data_as(C.c_void_p), blob.size, C.byref(h)))
        self.h = h
        ctx._retain()

    def __del__(self):
        if getattr(self, "h", None):
            self.ctx.lib.mlip_model_destroy(self.h)
            self.h = None
            self.ctx._release()


class Graph:
    """mlip_build_graph: pos [N,3] float64 CUDA tensor, cell [3,3] host array, species int32 CUDA tensor."""

    def __init__(self, ctx: Context, pos, cell, species, r_cut: float):
        torch = _torch()
        assert pos.is_cuda and pos.dtype == torch.float64 and pos.is_contiguous()
        assert species.is_cuda and species.dtype == torch.int32 and species.is_contiguous()
        self.ctx = ctx
        self.n_atoms = int(pos.shape[0])
        cell = np.ascontiguousarray(cell, dtype=np.float64)
        h = C.c_void_p()
        ctx.check(ctx.lib.mlip_build_graph(ctx.h, C.c_void_p(pos.data_ptr()), cell.ctypes.data_as(C.c_void_p),
                                           C.c_void_p(species.data_ptr()), self.n_atoms, float(r_cut), C.byref(h)))
        self.h = h
        ctx._retain()
        n = C.c_int64()
        ctx.check(ctx.lib.mlip_graph_num_edges(self.h, C.byref(n)))
        self.num_edges = int(n.value)

    def export_edges(self):
        torch = _torch()
        dev = f"cuda:{self.ctx.device}"
        recv = torch.empty(self.num_edges, dtype=torch.int32, device=dev)
        send = torch.empty(self.num_edges, dtype=torch.int32, device=dev)
        shift = torch.empty((self.num_edges, 3), dtype=torch.int32, device=dev)
        self.ctx.check(self.ctx.lib.mlip_graph_export_edges(self.ctx.h, self.h, C.c_void_p(recv.data_ptr()),
                                                            C.c_void_p(send.data_ptr()), C.c_void_p(shift.data_ptr())))
        return recv, send, shift

    def __del__(self):
        if getattr(self, "h", None):
            self.ctx.lib.mlip_graph_destroy(self.h)
            self.h = None
            self.ctx._release()


class Partition:
    """mlip_partition (n_sub slabs), mlip_partition_grid (grid=(gx,gy,gz)) or, with n_shards > 1, mlip_partition_grid_shard
    (only the sub-domains k with k mod n_shards == shard are built)."""

    def __init__(self, ctx: Context, graph: Graph, halo: float, n_sub: int | None = None, grid=None, shard: int = 0,
                 n_shards: int = 1):
        self.ctx = ctx
        self.graph = graph
        h = C.c_void_p()
        if grid is not None and n_shards > 1:
            g = (C.c_int * 3)(*[int(x) for x in grid])
            ctx.check(ctx.lib.mlip_partition_grid_shard(ctx.h, graph.h, g, float(halo), int(shard), int(n_shards), C.byref(h)))
        elif grid is not None:
            g = (C.c_int * 3)(*[int(x) for x in grid])
            ctx.check(ctx.lib.mlip_partition_grid(ctx.h, graph.h, g, float(halo), C.byref(h)))
        else:
            ctx.check(ctx.lib.mlip_partition(ctx.h, graph.h, int(n_sub), float(halo), C.byref(h)))
        self.h = h
        ctx._retain()

    def info(self):
        n = C.c_int()
        self.ctx.check(self.ctx.lib.mlip_part_count(self.h, C.byref(n)))
        out = []
        for s in range(n.value):
            a, b, c = C.c_int64(), C.c_int64(), C.c_int64()
            self.ctx.check(self.ctx.lib.mlip_part_info(self.h, s, C.byref(a), C.byref(b), C.byref(c)))
            out.append(dict(n_owned=a.value, n_ext=b.value, n_edges=c.value))
        return out

    def layer_info(self, L: int):
        """mlip_part_layer_info for every sub-domain and layer -> [[dict(n_recv, n_send, n_edges)] * L] * n_sub."""
        n = C.c_int()
        self.ctx.check(self.ctx.lib.mlip_part_count(self.h, C.byref(n)))
        out = []
        for s in range(n.value):
            rows = []
            for l in range(L):
                a, b, c = C.c_int64(), C.c_int64(), C.c_int64()
                self.ctx.check(self.ctx.lib.mlip_part_layer_info(self.h, s, int(L), l, C.byref(a), C.byref(b), C.byref(c)))
                rows.append(dict(n_recv=a.value, n_send=b.value, n_edges=c.value))
            out.append(rows)
        return out

    def __del__(self):
        if getattr(self, "h", None):
            self.ctx.lib.mlip_part_destroy(self.h)
            self.h = None
            self.ctx._release()


def energy_forces(ctx: Context, model: Model, L: int, graph: Graph, part: Partition | None = None,
                  precision: int = MLIP_FP32, want_atom_energy: bool = True, out=None):
    """mlip_energy_forces -> (E float64[1], F float32[N,3], E_i float32[N] or None), CUDA tensors (async)."""
    torch = _torch()
    dev = f"cuda:{ctx.device}"
    if out is None:
        E = torch.empty(1, dtype=torch.float64, device=dev)
        F = torch.empty((graph.n_atoms, 3), dtype=torch.float32, device=dev)
        Ei = torch.empty(graph.n_atoms, dtype=torch.float32, device=dev) if want_atom_energy else None
    else:
        E, F, Ei = out
    ctx.check(ctx.lib.mlip_energy_forces(ctx.h, model.h, int(L), graph.h, part.h if part is not None else None,
                                         int(precision), C.c_void_p(E.data_ptr()), C.c_void_p(F.data_ptr()),
                                         C.c_void_p(Ei.data_ptr()) if Ei is not None else None))
    return E, F, Ei


def energy_forces_shard(ctx: Context, model: Model, L: int, graph: Graph, part: Partition, shard: int, n_shards: int,
                        precision: int = MLIP_FP32, want_atom_energy: bool = False, out=None):
    """mlip_energy_forces_shard -> this shard's partial (E, F, E_i); sum over shards = full result."""
    torch = _torch()
    dev = f"cuda:{ctx.device}"
    if out is None:
        E = torch.empty(1, dtype=torch.float64, device=dev)
        F = torch.empty((graph.n_atoms, 3), dtype=torch.float32, device=dev)
        Ei = torch.empty(graph.n_atoms, dtype=torch.float32, device=dev) if want_atom_energy else None
    else:
        E, F, Ei = out
    ctx.check(ctx.lib.mlip_energy_forces_shard(ctx.h, model.h, int(L), graph.h, part.h, int(shard), int(n_shards),
                                               int(precision), C.c_void_p(E.data_ptr()), C.c_void_p(F.data_ptr()),
                                               C.c_void_p(Ei.data_ptr()) if Ei is not None else None))
    return E, F, Ei


def energy_forces_stress(ctx: Context, model: Model, L: int, graph: Graph, part: Partition | None = None,
                         precision: int = MLIP_FP32, shard: int = 0, n_shards: int = 1):
    """mlip_energy_forces_stress -> (E float64[1], F float32[N,3], E_i float32[N], sigma float64[3,3]), CUDA tensors."""
    torch = _torch()
    dev = f"cuda:{ctx.device}"
    E = torch.empty(1, dtype=torch.float64, device=dev)
    F = torch.empty((graph.n_atoms, 3), dtype=torch.float32, device=dev)
    Ei = torch.empty(graph.n_atoms, dtype=torch.float32, device=dev)
    S = torch.empty((3, 3), dtype=torch.float64, device=dev)
    ctx.check(ctx.lib.mlip_energy_forces_stress(ctx.h, model.h, int(L), graph.h, part.h if part is not None else None,
                                                int(shard), int(n_shards), int(precision), C.c_void_p(E.data_ptr()),
                                                C.c_void_p(F.data_ptr()), C.c_void_p(Ei.data_ptr()),
                                                C.c_void_p(S.data_ptr())))
    return E, F, Ei, S


def md_nve(ctx: Context, model: Model, L: int, pos, vel, mass, cell: np.ndarray, species, dt: float, n_steps: int,
           grid=(1, 1, 1), halo: float = 0.0, precision: int = MLIP_FP32):
    """mlip_md_nve: pos/vel float64 CUDA tensors updated in place; returns total energy per step (numpy [n_steps+1])."""
    torch = _torch()
    assert pos.is_cuda and pos.dtype == torch.float64 and pos.is_contiguous()
    assert vel.is_cuda and vel.dtype == torch.float64 and vel.is_contiguous()
    assert mass.is_cuda and mass.dtype == torch.float64 and species.dtype == torch.int32
    cell = np.ascontiguousarray(cell, dtype=np.float64)
    g = (C.c_int * 3)(*[int(x) for x in grid])
    out = np.zeros(n_steps + 1, dtype=np.float64)
    ctx.check(ctx.lib.mlip_md_nve(ctx.h, model.h, int(L), C.c_void_p(pos.data_ptr()), C.c_void_p(vel.data_ptr()),
                                  C.c_void_p(mass.data_ptr()), cell.ctypes.data_as(C.c_void_p),
                                  C.c_void_p(species.data_ptr()), int(pos.shape[0]), g, float(halo), int(precision),
                                  float(dt), int(n_steps), out.ctypes.data_as(C.c_void_p)))
    return out


def md_run(ctx: Context, model: Model, L: int, pos, vel, mass, cell: np.ndarray, species, dt: float, n_steps: int,
           grid=(1, 1, 1), halo: float = 0.0, precision: int = MLIP_FP32, thermostat: int = MLIP_MD_NVE,
           temperature: float = 0.0, friction: float = 0.0, seed: int = 0, skin: float = 0.0, cuda_graph: bool = False):
    """mlip_md_run: pos/vel float64 CUDA tensors updated in place; returns (total energy per step [n_steps+1], stats dict)."""
    torch = _torch()
    assert pos.is_cuda and pos.dtype == torch.float64 and pos.is_contiguous()
    assert vel.is_cuda and vel.dtype == torch.float64 and vel.is_contiguous()
    assert mass.is_cuda and mass.dtype == torch.float64 and species.dtype == torch.int32
    cell = np.ascontiguousarray(cell, dtype=np.float64)
    g = (C.c_int * 3)(*[int(x) for x in grid])
    out = np.zeros(n_steps + 1, dtype=np.float64)
    prm = mlip_md_params(float(dt), int(n_steps), int(thermostat), float(temperature), float(friction), int(seed),
                         float(skin), 1 if cuda_graph else 0, 0)
    st = mlip_md_stats()
    ctx.check(ctx.lib.mlip_md_run(ctx.h, model.h, int(L), C.c_void_p(pos.data_ptr()), C.c_void_p(vel.data_ptr()),
                                  C.c_void_p(mass.data_ptr()), cell.ctypes.data_as(C.c_void_p),
                                  C.c_void_p(species.data_ptr()), int(pos.shape[0]), g, float(halo), int(precision),
                                  C.byref(prm), out.ctypes.data_as(C.c_void_p), C.byref(st)))
    return out, dict(n_rebuilds=int(st.n_rebuilds), n_graph_replays=int(st.n_graph_replays), ms_total=float(st.ms_total))


MLIP_SCAN_NOALLOC_MAX = 67108864


def _scan(fn, ctx: Context, values, out):
    torch = _torch()
    assert values.is_cuda and values.dtype == torch.int32 and values.is_contiguous()
    n = values.numel()
    if out is None:
        out = torch.empty(n + 1, dtype=torch.int32, device=values.device)
    assert out.is_cuda and out.dtype == torch.int32 and out.is_contiguous() and out.numel() >= n + 1
    ctx.check(fn(ctx.h, C.c_void_p(values.data_ptr() if n else 0), C.c_void_p(out.data_ptr()), n))
    return out


def scan_i32(ctx: Context, values, out=None):
    """mlip_scan_i32: exclusive prefix sum (n + 1 entries, the last is the total) through the allocating path."""
    return _scan(ctx.lib.mlip_scan_i32, ctx, values, out)


def scan_i32_noalloc(ctx: Context, values, out=None):
    """mlip_scan_i32_noalloc: the same with a fixed device scratch array, no allocation inside the call (pass `out` to
    keep the binding allocation-free too); n <= MLIP_SCAN_NOALLOC_MAX."""
    return _scan(ctx.lib.mlip_scan_i32_noalloc, ctx, values, out)


def step_host(ctx: Context, model: Model, L: int, pos: np.ndarray, cell: np.ndarray, species: np.ndarray,
              grid=(1, 1, 1), halo: float = 0.0, precision: int = MLIP_FP32, forces_out: np.ndarray | None = None):
    """mlip_step_host: whole step from host arrays (pinned or pageable); returns (E float, F [N,3] float32)."""
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    cell = np.ascontiguousarray(cell, dtype=np.float64)
    species = np.ascontiguousarray(species, dtype=np.int32)
    n = pos.shape[0]
    F = forces_out if forces_out is not None else np.empty((n, 3), dtype=np.float32)
    E = np.zeros(1, dtype=np.float64)
    g = (C.c_int * 3)(*[int(x) for x in grid])
    ctx.check(ctx.lib.mlip_step_host(ctx.h, model.h, int(L), pos.ctypes.data_as(C.c_void_p), cell.ctypes.data_as(C.c_void_p),
                                     species.ctypes.data_as(C.c_void_p), n, g, float(halo), int(precision),
                                     E.ctypes.data_as(C.c_void_p), F.ctypes.data_as(C.c_void_p)))
    return float(E[0]), F
