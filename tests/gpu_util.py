"""Helpers shared by the -m gpu parity tests (calls go through the C ABI via the ctypes binding)."""
import numpy as np
import torch

import oracle
import synth
import paper_2312_06838_b200 as gnn


def dev(x, dtype=None):
    t = torch.from_numpy(np.ascontiguousarray(x))
    if dtype is not None:
        t = t.to(dtype)
    return t.cuda()


def make_model(arch, weights, precision=gnn.FP32_VALIDATION, max_batch_jets=1024, slices=1, max_particles=None):
    return gnn.Model(gnn.arch_struct(arch, max_batch_jets=max_batch_jets, precision=precision,
                                     workspace_slices=slices, max_particles=max_particles), weights)


def run_ragged(model, batch):
    f, c, o = dev(batch.feats), dev(batch.coords), dev(batch.offsets)
    out = model.infer(f, c, o)
    torch.cuda.synchronize()
    return out.cpu().numpy().astype(np.float64)


def ambiguous_points(dk, dk1, rel=1e-5):
    """R21: point is ambiguous iff (d^(k+1) - d^(k)) / d^(k+1) < rel on the ORACLE's distances (d^(k+1) = 0 -> ambiguous)."""
    with np.errstate(divide="ignore", invalid="ignore"):
        gap = (dk1 - dk) / dk1
    amb = np.where(np.isfinite(dk1), (dk1 == 0) | (gap < rel), False)
    return amb


def compare_sets(idx_gpu, idx_orc, amb):
    """Returns (#non-ambiguous points whose sets differ, #ambiguous points whose sets differ, mask of differing points)."""
    a = np.sort(idx_gpu, axis=1)
    b = np.sort(idx_orc, axis=1)
    diff = (a != b).any(axis=1)
    return int((diff & ~amb).sum()), int((diff & amb).sum()), diff


def staged_fp32(model, arch, weights, batch):
    """End-to-end through the per-stage entry points (the same kernels the forward uses), checking neighbour sets
    block by block against the oracle's dumps.  Returns (logits, per-block bad/ambiguous-flip counts, excluded jets)."""
    r = oracle.forward(arch, weights, batch.feats, batch.coords, batch.offsets, dumps=True)
    o = dev(batch.offsets)
    x = dev(batch.feats)
    space = dev(batch.coords)
    report = []
    excluded = np.zeros(batch.n_jets, bool)
    jet_of = np.repeat(np.arange(batch.n_jets), batch.counts())
    for l in range(len(arch.channels)):
        idx = model.debug_knn(space, o, arch.k)
        torch.cuda.synchronize()
        amb = ambiguous_points(r["dk"][l], r["dk1"][l])
        bad, flips, diff = compare_sets(idx.cpu().numpy(), r["nbr"][l], amb)
        report.append((bad, flips))
        excluded[np.unique(jet_of[diff & amb])] = True
        x = model.debug_edgeconv(l, x, idx, o)
        space = x
    logits = model.debug_pool_head(x, o)
    torch.cuda.synchronize()
    return logits.cpu().numpy().astype(np.float64), r, report, excluded
