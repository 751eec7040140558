"""Helpers for the -m gpu parity tests: run the CUDA path through the C ABI binding and the
float64 oracle on the same seeded inputs, and the error metrics of reading R14."""
import numpy as np

from oracle import mlip_oracle as O


def rms(x):
    return float(np.sqrt(np.mean(np.square(x))))


def oracle_model(spec, blob):
    return O.parse_weights(spec.n_species, spec.d, spec.n_rbf, spec.L_max, spec.r_cut, spec.agg_scale, blob,
                           r_cut3=getattr(spec, "r_cut3", 0.0))


def gpu_setup(spec, blob):
    import paper_2509_21694_b200 as mlip
    ctx = mlip.Context(0)
    model = mlip.Model(ctx, spec.n_species, spec.d, spec.n_rbf, spec.L_max, spec.r_cut, spec.agg_scale, blob,
                       r_cut3=getattr(spec, "r_cut3", 0.0))
    return mlip, ctx, model


def gpu_graph(mlip, ctx, system, r_cut):
    import torch
    pos = torch.tensor(system.pos, dtype=torch.float64, device="cuda:0").contiguous()
    species = torch.tensor(system.species, dtype=torch.int32, device="cuda:0").contiguous()
    return mlip.Graph(ctx, pos, system.cell, species, r_cut)


def gpu_energy_forces(mlip, ctx, model, L, graph, part=None, precision=0):
    import torch
    E, F, Ei = mlip.energy_forces(ctx, model, L, graph, part, precision)
    ctx.status()   # synchronises; raises MlipError for a device-side error (e.g. MLIP_ERR_NUMERIC)
    return float(E.item()), F.cpu().numpy().astype(np.float64), Ei.cpu().numpy().astype(np.float64)


def errors(E, F, Ei, E_ref, F_ref, Ei_ref):
    """eps_E = |E - E_ref| / sum_i |E_i,ref| ; rel_Ei = max_i |E_i - E_i,ref| / max(|E_i,ref|, RMS(E_ref)) (the
    per-atom energy relative error of north_star, reading R14: a readout or ownership error that preserves the sum does
    not cancel in it) ; max force error / RMS(F_ref) ; RMS force error / RMS(F_ref)"""
    return dict(eps_E=abs(E - E_ref) / np.abs(Ei_ref).sum(),
                rel_Ei=float((np.abs(Ei - Ei_ref) / np.maximum(np.abs(Ei_ref), max(rms(Ei_ref), 1e-30))).max()),
                max_Ei=np.abs(Ei - Ei_ref).max() / max(rms(Ei_ref), 1e-30),
                max_F=np.abs(F - F_ref).max() / max(rms(F_ref), 1e-30),
                rms_F=rms(F - F_ref) / max(rms(F_ref), 1e-30))
