"""-m gpu parity of the BDT kernel (csrc/bdt.cu) against oracle/bdt.py: the reached leaves are decided
by fp32 comparisons on both sides (identical decisions), the margin is an fp32 sum of <= 100 terms of |leaf| ~ 0.1 against
the oracle's fp64 sum, so probabilities agree to a few fp32 ulps: 2e-6 absolute."""
import numpy as np
import pytest
import torch

import synth
import paper_2312_06838_b200 as gnn
from oracle import bdt as obdt

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("depth,T,F,N", [(6, 100, 20, 100003), (1, 5, 3, 1000), (3, 17, 7, 257), (8, 40, 20, 5000), (6, 100, 20, 1)])
def test_bdt_against_oracle(depth, T, F, N):
    f, t, l = synth.make_bdt(seed=depth * 10 + T, n_trees=T, depth=depth, n_features=F)
    x = synth.make_bdt_events(N, F, seed=N)
    if N > 100:
        x[::31, 1] = np.nan                              # NaN goes right
        x[5, :] = t[0, 0]                                 # equality goes right
    m = gnn.Bdt(f, t, l, F)
    out = m.infer(torch.from_numpy(x).cuda()).cpu().numpy().astype(np.float64)
    ref = obdt.predict(f, t, l, x)
    assert np.abs(out - ref).max() < 2e-6
    h = torch.empty((N, 2), dtype=torch.float32).pin_memory()
    m.infer_host(torch.from_numpy(x).pin_memory(), h)
    assert np.array_equal(h.numpy(), out.astype(np.float32))
    m.close()


def test_bdt_argument_checks():
    f, t, l = synth.make_bdt(n_trees=4, depth=3, n_features=5)
    with pytest.raises(gnn.GnnError):
        gnn.Bdt(f, t, l, 3)                               # feature index out of range
    f2, t2, l2 = synth.make_bdt(n_trees=2000, depth=8, n_features=5)
    with pytest.raises(gnn.GnnError):
        gnn.Bdt(f2, t2, l2, 5)                            # forest larger than one SM's shared memory
    m = gnn.Bdt(f, t, l, 5)
    assert m.infer(torch.empty((0, 5), device="cuda")).shape == (0, 2)
    m.close()


def test_a_later_smaller_forest_does_not_break_an_earlier_larger_one():
    """The dynamic-shared-memory cap is an attribute of the kernel on the device, not of one forest: creating a small forest
    after a large one must leave the large one launchable (the cap is always raised to the 200 KB ceiling)."""
    fb, tb, lb = synth.make_bdt(seed=71, n_trees=100, depth=6, n_features=20)        # ~ 130 KB of shared memory
    fs, ts, ls = synth.make_bdt(seed=72, n_trees=3, depth=2, n_features=4)           # a few KB
    x = synth.make_bdt_events(3000, 20, seed=73)
    big = gnn.Bdt(fb, tb, lb, 20)
    small = gnn.Bdt(fs, ts, ls, 4)
    xs = synth.make_bdt_events(100, 4, seed=74)
    assert np.abs(small.infer(torch.from_numpy(xs).cuda()).cpu().numpy() - obdt.predict(fs, ts, ls, xs)).max() < 2e-6
    out = big.infer(torch.from_numpy(x).cuda())
    torch.cuda.synchronize()
    assert np.abs(out.cpu().numpy().astype(np.float64) - obdt.predict(fb, tb, lb, x)).max() < 2e-6
    # rows are stored as float2: an output pointer that is not 8-byte aligned is refused, not written through
    buf = torch.empty(2 * 3000 + 1, dtype=torch.float32, device="cuda")
    with pytest.raises(gnn.GnnError):
        big.infer(torch.from_numpy(x).cuda(), out=buf[1:].view(3000, 2))
    big.close(); small.close()
