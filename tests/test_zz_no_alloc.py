"""-m gpu test of gnn_knn_noalloc, the one entry point of libgnn.so that allocates no device memory.

Some users of this library run where cudaMalloc is off limits: a plugin inside an application that owns the device heap and
hands out fixed buffers, a real-time loop that must not wait on the allocator's device-wide lock, a process whose GPU memory
was budgeted to the byte before the library was loaded.  They cannot create a gnn_model (gnn_create allocates), so
gnn_knn_noalloc runs the exact kNN step on the caller's buffers alone and keeps its intermediate data in a fixed array inside
libgnn.so (limits: 1024 jets / 8192 particles per call; calls share that array and must not overlap on the GPU).

Checked here, through the C ABI: its neighbour indices are IDENTICAL (integer work: bit-exact, the bar of the other kNN
tests) to gnn_debug_knn's on a GNN_FP32_VALIDATION model -- the existing path, whose scratch is the model's cudaMalloc'ed
workspace -- on two calls in a row.  The second call is a different, smaller batch in another space, so anything the first
call left in the shared array would show up as a difference.  Also: sizes beyond the limits are refused.

This file sorts after every other test file on purpose (pytest -x stops at the first failure); it needs nothing from the
tests before it and passes alone in a fresh process as well.
"""
import numpy as np
import pytest
import torch

import synth
import paper_2312_06838_b200 as gnn
from gpu_util import dev, make_model

pytestmark = pytest.mark.gpu


def spaces():
    """(space [N, D], offsets) pairs: coordinates of ragged jets (D = 2: distances computed inside the selection) and a
    64-dimensional feature-like space (D = 64: distances staged through the scratch matrix), ragged sizes with a tail."""
    b1 = synth.make_particlenet_batch(seed=4101, n_jets=160)            # ~6400 particles, n in [5, 100]
    rng = np.random.default_rng(4102)
    b2 = synth.make_edge_case_batch(F=4, seed=4103)                     # n = 0, 1, 2, ..., 127, 128
    feat = rng.standard_normal((b1.n_particles, 64)).astype(np.float32)
    feat2 = rng.standard_normal((b2.n_particles, 64)).astype(np.float32)
    return [(feat, b1.offsets), (b2.coords.astype(np.float32), b2.offsets), (feat2, b2.offsets), (b1.coords.astype(np.float32), b1.offsets)]


def test_noalloc_knn_equals_the_model_path_on_consecutive_calls():
    a = synth.ARCHS["particlenet"]
    model = make_model(a, synth.make_weights(a), precision=gnn.FP32_VALIDATION, max_batch_jets=1024, max_particles=128)
    k = a.k
    cases = spaces()
    # existing path first (its own workspace), results kept on the host
    want = []
    for space, off in cases:
        idx = model.debug_knn(dev(space), dev(off), k)
        torch.cuda.synchronize()
        assert model.status_check() == 0
        want.append(idx.cpu().numpy())
    # the no-allocation entry: back-to-back calls on one stream, outputs into buffers made beforehand, read afterwards
    ins = [(dev(space), dev(off)) for space, off in cases]
    outs = [torch.full((space.shape[0], k), -7, dtype=torch.int32, device="cuda") for space, _ in cases]
    torch.cuda.synchronize()
    for (sp, off), out in zip(ins, outs):
        gnn.knn_noalloc(sp, off, k, max_particles=128, idx=out)
    torch.cuda.synchronize()
    for i, (out, ref) in enumerate(zip(outs, want)):
        got = out.cpu().numpy()
        assert got.shape == ref.shape
        assert (got != -7).all(), "case %d: rows left unwritten" % i
        assert np.array_equal(got, ref), "case %d: %d of %d entries differ" % (i, int((got != ref).sum()), ref.size)
    model.close()


def test_noalloc_knn_needs_no_model_and_repeats_itself():
    """Alone in the process (no gnn_create anywhere): same input twice -> same output, and it agrees with a numpy brute force
    on integer lattice points, where fp32 distances are exact and ties fall to the lower index."""
    rng = np.random.default_rng(4104)
    sizes = [1, 7, 33, 128, 2, 64]
    off = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int32)
    pts = rng.integers(-6, 7, size=(off[-1], 3)).astype(np.float32)
    k = 8
    sp, o = dev(pts), dev(off)
    a = gnn.knn_noalloc(sp, o, k).cpu().numpy()
    b = gnn.knn_noalloc(sp, o, k).cpu().numpy()
    assert np.array_equal(a, b)
    for j, n in enumerate(sizes):
        p = pts[off[j]:off[j + 1]].astype(np.int64)
        d = ((p[:, None, :] - p[None, :, :]) ** 2).sum(-1)
        for i in range(n):
            cand = [c for c in np.lexsort((np.arange(n), d[i])) if c != i][:k]
            ref = np.full(k, -1)
            ref[:len(cand)] = cand
            assert np.array_equal(a[off[j] + i], ref), (j, i)


def test_noalloc_knn_refuses_what_does_not_fit():
    off = dev(np.array([0, 4], np.int32))
    sp = dev(np.zeros((4, 2), np.float32))
    idx = torch.zeros((4, 4), dtype=torch.int32, device="cuda")
    L = gnn.lib()
    import ctypes as C
    s = C.c_void_p(torch.cuda.current_stream().cuda_stream)
    p = lambda t: C.c_void_p(t.data_ptr())
    assert L.gnn_knn_noalloc(p(sp), 2, p(off), 1025, 4, 128, 4, p(idx), s) == -4      # GNN_ERR_BATCH_TOO_LARGE: jets
    assert L.gnn_knn_noalloc(p(sp), 2, p(off), 1, 8193, 128, 4, p(idx), s) == -4      # ... particles
    assert L.gnn_knn_noalloc(p(sp), 2, p(off), 1, 4, 129, 4, p(idx), s) == -8         # GNN_ERR_BAD_ARG: max_particles
    assert L.gnn_knn_noalloc(p(sp), 2, p(off), 1, 4, 128, 4, p(idx), s) == 0
    torch.cuda.synchronize()
    assert np.array_equal(idx.cpu().numpy(), np.array([[1, 2, 3, -1], [0, 2, 3, -1], [0, 1, 3, -1], [0, 1, 2, -1]]))
