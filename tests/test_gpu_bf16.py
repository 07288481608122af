"""-m gpu parity tests, GNN_BF16 production mode: the tcgen05 EdgeConv path against the fp64 oracle, through the C ABI.
Bar (BASELINE.json north_star): logits within 5e-2 absolute of the oracle on every jet, argmax agreement >= 99.9 %.
No neighbour-set bar exists in this mode (R20); the flip rate is only reported."""
import numpy as np
import pytest
import torch

import oracle
import synth
import paper_2312_06838_b200 as gnn
from gpu_util import dev, make_model, run_ragged

pytestmark = pytest.mark.gpu
LOGIT_TOL = 5e-2
ARGMAX_MIN = 0.999


def bf16_model(name, max_batch_jets=1024, **kw):
    a = synth.ARCHS[name]
    w = synth.make_weights(a)
    return a, w, make_model(a, w, precision=gnn.BF16, max_batch_jets=max_batch_jets, **kw)


@pytest.fixture(scope="module")
def pn():
    return bf16_model("particlenet", 4096)


def check_logits(lg, ref):
    err = np.abs(lg - ref).max(1)
    assert err.max() < LOGIT_TOL, "max |dlogit| = %.3e" % err.max()
    agree = (np.argmax(lg, 1) == np.argmax(ref, 1)).mean()
    assert agree >= ARGMAX_MIN, "argmax agreement %.4f" % agree
    return err


# ---- EdgeConv stage: the fused tcgen05 kernel given the oracle's neighbour indices ----------------------------------
@pytest.mark.parametrize("name,block", [("tiny", 0), ("particlenet", 0), ("particlenet", 1), ("particlenet", 2)])
def test_edgeconv_stage_given_oracle_indices(name, block):
    """Sizes span several 128-row MMA tiles, a ragged last tile, jets with k_eff < k (n = 1, 2, 5, 16) and n = 128."""
    a, w, m = bf16_model(name, 64)
    rng = np.random.default_rng(block)
    counts = [16] * 5 if name == "tiny" else [1, 2, 17, 40, 100, 5, 16, 61, 40, 40, 33, 128, 3]
    off = np.zeros(len(counts) + 1, np.int32); off[1:] = np.cumsum(counts)
    x = rng.normal(0, 1, (off[-1], a.block_in(block))).astype(np.float32)
    if block > 0:
        x = np.maximum(x, 0)                                   # block inputs after block 1 are post-ReLU
    idx, _, _ = oracle.knn(x, off, a.k)
    y = m.debug_edgeconv(block, dev(x), dev(idx), dev(off)).cpu().numpy()
    ref = oracle.edgeconv(a, w, block, x, idx, off)
    err = np.abs(y - ref)
    # operands of the three edge-MLP GEMMs are bf16 (2^-9 relative each), accumulators fp32: the error of one output
    # is a few 1e-3 of the largest activation feeding it
    assert err.max() < 6e-3 * max(1.0, np.abs(ref).max())
    assert err.mean() < 5e-4 * max(1.0, np.abs(ref).max())
    m.close()


@pytest.mark.parametrize("k", [1, 2, 8, 32])
def test_edgeconv_stage_other_k(k):
    """Neighbour counts other than the configs' 16 and 4 take the runtime-k path of the gather and, for k = 32, the
    extra fp32 step of the E3 row reduction; blocks with C = 64 (SIMT pre kernel) and C = 128 (tcgen05 tf32 pre kernel)."""
    a = synth.Arch(in_features=6, k=k, channels=((64, 64, 64), (128, 128, 128)), fc_hidden=(32,), max_particles=64)
    w = synth.make_weights(a)
    m = make_model(a, w, precision=gnn.BF16, max_batch_jets=32)
    rng = np.random.default_rng(100 + k)
    counts = [1, 2, 3, 9, 33, 40, 64, 17, 5, 40, 64, 31]
    off = np.zeros(len(counts) + 1, np.int32); off[1:] = np.cumsum(counts)
    for block in (0, 1):
        x = rng.normal(0, 1, (off[-1], a.block_in(block))).astype(np.float32)
        if block > 0:
            x = np.maximum(x, 0)
        idx, _, _ = oracle.knn(x, off, a.k)
        y = m.debug_edgeconv(block, dev(x), dev(idx), dev(off)).cpu().numpy()
        ref = oracle.edgeconv(a, w, block, x, idx, off)
        err = np.abs(y - ref)
        assert err.max() < 6e-3 * max(1.0, np.abs(ref).max()), (k, block, err.max())
    m.close()


# ---- whole network -----------------------------------------------------------------------------------------------------
def test_tiny_end_to_end():
    a, w, m = bf16_model("tiny", 64)
    t = synth.make_tiny()
    lg = run_ragged(m, t)
    ref = oracle.forward(a, w, t.feats, t.coords, t.offsets)
    check_logits(lg, ref)
    assert (np.argmax(lg, 1) == np.argmax(ref, 1)).all()       # R22: 32 / 32
    m.close()


def test_particlenet_full_batch_1024(pn, record_property):
    """BASELINE configs[1] at its full size, in the launch configuration bench.py times (one gnn_infer)."""
    a, w, m = pn
    b = synth.make_particlenet_batch()
    lg = run_ragged(m, b)
    assert m.status_check() == 0
    r = oracle.forward(a, w, b.feats, b.coords, b.offsets, dumps=True)
    ref = r["logits"]
    err = check_logits(lg, ref)
    assert err.mean() < 2.5e-2
    # ---- parity protocol of SURVEY 8(c) for this mode (R20, R22): reported, not enforced.  Per-block neighbour flip rate =
    # share of the points whose neighbour SET, computed by the production kNN on the GPU's own block input, differs from the
    # oracle's set on the oracle's input (it contains the upstream bf16 noise); and the oracle's logit-gap histogram, which
    # says how many jets sit close enough to the decision boundary for a 5e-2 logit error to flip their argmax.
    o = dev(b.offsets)
    x, space, flips = dev(b.feats), dev(b.coords), []
    for l in range(len(a.channels)):
        idx = m.debug_knn(space, o, a.k)
        gi, oi = np.sort(idx.cpu().numpy(), 1), np.sort(r["nbr"][l], 1)
        flips.append(float((gi != oi).any(1).mean()))
        x = m.debug_edgeconv(l, x, idx, o)
        space = x
    staged = m.debug_pool_head(x, o).cpu().numpy().astype(np.float64)
    assert np.abs(staged - lg).max() < 5e-3                 # same kernels up to the pooling route (stored block output vs fused sums)
    gap = np.abs(ref[:, 1] - ref[:, 0])
    edges = [0.0, 0.05, 0.1, 0.2, 0.5, 1.0, 2.0, 5.0, np.inf]
    hist = np.histogram(gap, edges)[0].tolist()
    print("bf16 B=1024: max |dlogit| %.3e, mean %.3e; neighbour-set flip rate per block %s; oracle |z1 - z0| histogram over edges %s: %s"
          % (err.max(), err.mean(), ["%.4f" % f for f in flips], edges, hist))
    record_property("flip_rate_per_block", flips)
    record_property("oracle_logit_gap_histogram", {"edges": [str(e) for e in edges], "counts": hist})
    assert flips[0] < 2e-3 and max(flips) < 0.15            # block 1 is exact arithmetic on exact coordinates; later blocks carry bf16 noise


def test_ragged_4096_f9_sampled():
    """configs[2] at its full size (4096 jets, F = 9, CSR only); the oracle runs the first 1024 jets, which are
    compared inside the full batch (jets are independent)."""
    a, w, m = bf16_model("particlenet_f9", 4096)
    b = synth.make_ragged_batch()
    lg = run_ragged(m, b)
    assert m.status_check() == 0 and np.isfinite(lg).all()
    h = b.head(1024)
    ref = oracle.forward(a, w, h.feats, h.coords, h.offsets)
    check_logits(lg[:1024], ref)
    m.close()


def test_sweep_base_1024_sampled(pn):
    """configs[4] base arch at B = 1024 (P = 128, multiplicity ~ clip(Poisson(60),5,128)); oracle on the first 256."""
    a, w, m = pn
    b = synth.make_sweep_batch(n_jets=1024)
    lg = run_ragged(m, b)
    h = b.head(256)
    ref = oracle.forward(a, w, h.feats, h.coords, h.offsets)
    check_logits(lg[:256], ref)
    for B in (1, 16):                                          # nested batch sizes give the same jets
        assert np.array_equal(run_ragged(m, b.head(B)), lg[:B])


def test_sweep_base_16384_maximum_size():
    """configs[4] at its largest batch (16 384 jets, ~983 k particles, the workspace's maximum): finite logits, no device
    error, the first 256 jets within the parity bars of the oracle, and bitwise equal to the same jets run as a batch
    of 256 (batch-composition invariance at the size the sweep is timed at)."""
    a, w, m = bf16_model("particlenet", 16384)
    b = synth.make_sweep_batch(n_jets=16384)
    lg = run_ragged(m, b)
    assert m.status_check() == 0 and np.isfinite(lg).all()
    h = b.head(256)
    ref = oracle.forward(a, w, h.feats, h.coords, h.offsets)
    check_logits(lg[:256], ref)
    assert np.array_equal(run_ragged(m, h), lg[:256])
    m.close()


def test_sweep_wide_256_sampled():
    """configs[4] wide variant (EdgeConv channels 128, 256, 512, FC 512) at B = 256; the oracle runs all 256 jets (SURVEY 8(c):
    "first 256").  Block 3 (C = 512) takes the streamed-weight kernel, its stage is also checked alone."""
    a, w, m = bf16_model("wide", 256)
    b = synth.make_sweep_batch(n_jets=256)
    lg = run_ragged(m, b)
    assert m.status_check() == 0 and np.isfinite(lg).all()
    ref = oracle.forward(a, w, b.feats, b.coords, b.offsets)
    check_logits(lg, ref)
    rng = np.random.default_rng(7)
    counts = [1, 2, 17, 40, 100, 5, 16, 61, 128, 3]
    off = np.zeros(len(counts) + 1, np.int32); off[1:] = np.cumsum(counts)
    x = np.maximum(rng.normal(0, 1, (off[-1], a.block_in(2))), 0).astype(np.float32)
    idx, _, _ = oracle.knn(x, off, a.k)
    y = m.debug_edgeconv(2, dev(x), dev(idx), dev(off)).cpu().numpy()
    r2 = oracle.edgeconv(a, w, 2, x, idx, off)
    assert np.abs(y - r2).max() < 6e-3 * max(1.0, np.abs(r2).max())
    m.close()


def test_sweep_wide_4096_sampled():
    """configs[4] wide variant at B = 4096 (245 k particles: many tiles per CTA in every kernel, ragged tails); the oracle runs
    the first 256 jets, compared inside the full batch; nested batch sizes give the same jets bit for bit."""
    a, w, m = bf16_model("wide", 4096)
    b = synth.make_sweep_batch(n_jets=4096)
    lg = run_ragged(m, b)
    assert m.status_check() == 0 and np.isfinite(lg).all()
    h = b.head(256)
    ref = oracle.forward(a, w, h.feats, h.coords, h.offsets)
    check_logits(lg[:256], ref)
    assert np.array_equal(run_ragged(m, b.head(16)), lg[:16])
    m.close()


def test_edge_case_set(pn):
    a, w, m = pn
    b = synth.make_edge_case_batch(a.in_features)
    ref = oracle.forward(a, w, b.feats, b.coords, b.offsets)
    assert np.abs(run_ragged(m, b) - ref).max() < LOGIT_TOL
    for sizes in [(1,), (0,), (128,), (0, 0, 0), (2,), (17,)]:
        bb = synth.make_edge_case_batch(a.in_features, sizes=sizes)
        ref = oracle.forward(a, w, bb.feats, bb.coords, bb.offsets)
        assert np.abs(run_ragged(m, bb) - ref).max() < LOGIT_TOL
    d = synth.make_edge_case_batch(a.in_features, sizes=(20,))
    d.feats[10:] = d.feats[:10]; d.coords[10:] = d.coords[:10]   # duplicate particles: exact ties at d = 0
    ref = oracle.forward(a, w, d.feats, d.coords, d.offsets)
    assert np.abs(run_ragged(m, d) - ref).max() < LOGIT_TOL
    # |x| ~ 10 (as test_gpu_fp32's case): block 1's u and v are then O(10) terms that cancel in u_i + v_j, the worst case for
    # bf16 operands; the bar scales with the logits like the fp32 test's (5e-2 absolute at |logit| <= 1)
    big = synth.make_edge_case_batch(a.in_features, sizes=(40, 7, 100, 16), scale=10.0)
    ref = oracle.forward(a, w, big.feats, big.coords, big.offsets)
    lg = run_ragged(m, big)
    print("bf16 |x| ~ 10: max |dlogit| %.3e at max |logit| %.2f" % (np.abs(lg - ref).max(), np.abs(ref).max()))
    assert np.isfinite(lg).all() and np.abs(lg - ref).max() < LOGIT_TOL * max(1.0, np.abs(ref).max())


def test_batch_composition_invariance_is_bitwise(pn):
    """A jet's logits do not depend on its batch mates or its position (what makes dynamic batching legal, PAPER.md
    L53): MMA rows are independent and every reduction has a fixed order."""
    a, w, m = pn
    b = synth.make_particlenet_batch(n_jets=64)
    full = run_ragged(m, b)
    sel = [5, 2, 63, 7]
    assert np.array_equal(run_ragged(m, b.select(sel)), full[sel])


@pytest.mark.parametrize("P,interleave,garbage", [(100, False, np.nan), (128, True, 1e9)])
def test_padded_entry_is_padding_invariant(pn, P, interleave, garbage):
    a, w, m = pn
    b = synth.make_particlenet_batch(n_jets=48)
    ref = run_ragged(m, b)
    f, c, mk = synth.pad_batch(b, P, interleave=interleave, garbage=garbage)
    out = m.infer_padded(dev(f), dev(c), dev(mk))
    torch.cuda.synchronize()
    assert m.status_check() == 0
    assert np.array_equal(out.cpu().numpy().astype(np.float64), ref)


def test_device_side_errors_bf16():
    a, w, m = bf16_model("particlenet", 16, max_particles=100)
    b = synth.make_particlenet_batch(n_jets=4)
    off = b.offsets.copy(); off[2] = off[1] - 1
    out = m.infer(dev(b.feats), dev(b.coords), dev(off))
    torch.cuda.synchronize()
    assert torch.isnan(out).all() and m.status_check() == -6
    big = synth.make_edge_case_batch(a.in_features, sizes=(10, 101, 12))
    out = m.infer(dev(big.feats), dev(big.coords), dev(big.offsets)).cpu().numpy()
    assert m.status_check() == -7
    assert np.isnan(out[1]).all() and np.isfinite(out[[0, 2]]).all()
    m.close()


def test_batcher_bf16_equals_direct():
    a, w, m = bf16_model("particlenet", 1024, slices=2, max_particles=100)
    pool = synth.make_client_pool(1, n_requests=8)
    direct = [run_ragged(m, r) for r in pool]
    bt = gnn.Batcher(m, max_batch_jets=1024, max_queue_delay_us=1000, n_instances=2)
    tickets = [bt.submit(r.feats, r.coords, r.offsets) for r in pool]
    for (t, out), ref in zip(tickets, direct):
        rc, _, _ = bt.wait(t)
        assert rc == 0
        assert np.array_equal(out.astype(np.float64), ref)
    bt.close()
    m.close()


def test_forward_is_bitwise_repeatable_back_to_back(pn):
    """The forward runs on one stream with programmatic dependent launches (a kernel's prologue under its predecessor's tail,
    the pre kernel and the kNN of a block side by side; api.cu forward()).  Back-to-back forwards over batches of different
    sizes, with and without an L2 eviction in between, must reproduce their first result bit for bit: a missing dependency
    between two kernels shows up as a sporadic difference."""
    _, _, m = pn
    flush = torch.empty(160 << 20, dtype=torch.uint8, device="cuda")
    bs = []
    for r, B in enumerate((1024, 16, 1, 300, 77)):
        b = synth.make_particlenet_batch(seed=5000 + r, n_jets=B)
        bs.append((dev(b.feats), dev(b.coords), dev(b.offsets)))
    first = [None] * len(bs)
    for it in range(150):
        i = it % len(bs)
        if it % 3 == 0:
            flush.zero_()
        out = m.infer(*bs[i]).clone()
        if first[i] is None:
            first[i] = out
        else:
            assert torch.equal(out, first[i]), "forward %d (batch %d) differs from its first result" % (it, i)
    torch.cuda.synchronize()
    assert m.status_check() == 0


def test_host_entry_pipelined_equals_blocking():
    """gnn_infer_host_begin / _end with two slices in flight on two streams gives bitwise the logits of the blocking
    gnn_infer_host and of the device-resident gnn_infer; device-side errors come back from _end."""
    a = synth.ARCHS["particlenet"]
    w = synth.make_weights(a)
    m = make_model(a, w, precision=gnn.BF16, max_batch_jets=256, slices=2, max_particles=100)
    bs = [synth.make_particlenet_batch(seed=700 + i, n_jets=64 + 32 * i) for i in range(4)]
    hb = [tuple(torch.from_numpy(x).pin_memory() for x in (b.feats, b.coords, b.offsets)) for b in bs]
    ref = [run_ragged(m, b).astype(np.float32) for b in bs]
    outs = [torch.empty((b.n_jets, 2), dtype=torch.float32).pin_memory() for b in bs]
    st = [torch.cuda.Stream(), torch.cuda.Stream()]
    for i in range(4):
        if i >= 2:
            m.infer_host_end(stream=st[i & 1], slice=i & 1)
        m.infer_host_begin(*hb[i], outs[i], stream=st[i & 1], slice=i & 1)
    for sl in range(2):
        m.infer_host_end(stream=st[sl], slice=sl)
    for i in range(4):
        assert np.array_equal(outs[i].numpy(), ref[i])
        blocking = torch.empty_like(outs[i])
        m.infer_host(*hb[i], blocking)
        assert np.array_equal(blocking.numpy(), ref[i])
    bad = hb[0][2].clone(); bad[3] = bad[5] + 1                 # offsets not monotone
    m.infer_host_begin(hb[0][0], hb[0][1], bad.pin_memory(), outs[0], stream=st[0], slice=0)
    with pytest.raises(gnn.GnnError) as e:
        m.infer_host_end(stream=st[0], slice=0)
    assert e.value.code == -6                                   # GNN_ERR_BAD_OFFSETS
    m.infer_host_end(stream=st[0], slice=0)                     # nothing in flight: a no-op
    m.close()


def test_forward_in_a_callers_cuda_graph_and_graph_replay(pn):
    """include/gnn.h: the forward is enqueued on the caller's stream alone, so it can be captured into a CUDA graph of the
    caller's; and gnn_infer replays a graph of its own when a call's arguments repeat.  Both must read the CURRENT contents of
    the input buffers: the same buffers refilled with other jets (same B and N) give those jets' logits, bitwise equal to a
    first-time call on fresh buffers."""
    _, _, m = pn
    b1 = synth.make_particlenet_batch(seed=901, n_jets=48)
    # a second batch with the same multiplicities (hence the same B, N and offsets) but other particles
    b2 = synth.make_particlenet_batch(seed=902, n_jets=400)
    order = np.argsort(b2.counts(), kind="stable")
    picked, pool = [], list(order)
    for n in b1.counts():
        j = next((j for j in pool if b2.counts()[j] == n), None)
        if j is None:
            pytest.skip("no jet of matching multiplicity in the donor batch")
        pool.remove(j); picked.append(int(j))
    b2 = b2.select(picked)
    assert np.array_equal(b2.offsets, b1.offsets)
    ref1, ref2 = run_ragged(m, b1), run_ragged(m, b2)              # fresh buffers each: never a replay
    f, c, o = dev(b1.feats), dev(b1.coords), dev(b1.offsets)
    out = torch.empty((b1.n_jets, 2), dtype=torch.float32, device="cuda")
    for _ in range(3):                                             # third call: the library's own graph replay
        m.infer(f, c, o, logits=out)
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy().astype(np.float64), ref1)
    f.copy_(dev(b2.feats)); c.copy_(dev(b2.coords))
    m.infer(f, c, o, logits=out)                                   # replayed graph, new contents
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy().astype(np.float64), ref2)
    # the caller's own capture
    g = torch.cuda.CUDAGraph()
    out2 = torch.empty_like(out)
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        m.infer(f, c, o, logits=out2, stream=side)                 # warm (nothing lazy inside the capture)
        side.synchronize()
        with torch.cuda.graph(g, stream=side):
            m.infer(f, c, o, logits=out2, stream=side)
    torch.cuda.current_stream().wait_stream(side)
    f.copy_(dev(b1.feats)); c.copy_(dev(b1.coords))
    g.replay()
    torch.cuda.synchronize()
    assert np.array_equal(out2.cpu().numpy().astype(np.float64), ref1)
    assert m.status_check() == 0


def test_no_grouped_knn_anywhere_still_pools_correctly():
    """An architecture none of whose kNN spaces has a grouped kernel (5 coordinates; the later block's space is 32 wide), with
    k = 16 and C_last = 64, so the last edge kernel COULD pool in its epilogue.  That epilogue reads the particle -> jet map
    only the grouped kNN kernels write; the forward must notice that nobody wrote it and pool the stored block output instead
    (before the fix it scattered the sums through uninitialised jet ids).  Run twice: a second forward must not depend on
    what the first left behind."""
    a = synth.Arch(in_features=6, k=16, channels=((32, 32, 32), (64, 64, 64)), fc_hidden=(64,), coord_dims=5, max_particles=128)
    w = synth.make_weights(a)
    m = make_model(a, w, precision=gnn.BF16, max_batch_jets=64)
    rng = np.random.default_rng(515)
    counts = [1, 2, 17, 40, 100, 5, 16, 0, 61, 40, 33, 128, 3, 40]
    off = np.zeros(len(counts) + 1, np.int32); off[1:] = np.cumsum(counts)
    feats = rng.normal(0, 1, (off[-1], a.in_features)).astype(np.float32)
    coords = rng.normal(0, 0.3, (off[-1], a.coord_dims)).astype(np.float32)
    ref = oracle.forward(a, w, feats, coords, off)
    f, c, o = dev(feats), dev(coords), dev(off)
    for _ in range(2):
        lg = m.infer(f, c, o)
        torch.cuda.synchronize()
        assert m.status_check() == 0
        check_logits(lg.cpu().numpy().astype(np.float64), ref)
    m.close()
