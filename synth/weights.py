"""Random weight blobs.  PAPER.md L264: the served demo model "was left untrained with randomized weights".

Draw order is normative: one `default_rng(seed)` per architecture; per block, per
layer (in,out) in [(2*C_in,C1),(C1,C2),(C2,C3)]: W ~ N(0, 2/in) shape (out,in), scale ~ N(1,0.1), shift ~ N(0,0.1);
then the shortcut (C3, C_in) likewise; then per FC: W ~ N(0, 2/in), bias ~ N(0,0.1).  float64 draws, cast to fp32.
The concatenation order IS the blob layout of include/gnn.h.
"""
import numpy as np
from .arch import Arch, weight_count


def make_weights(a: Arch, seed: int = 0) -> np.ndarray:
    rng = np.random.default_rng(seed)
    parts = []
    for l, (c1, c2, c3) in enumerate(a.channels):
        cin = a.block_in(l)
        for (i, o) in ((2 * cin, c1), (c1, c2), (c2, c3)):
            parts.append(rng.normal(0.0, np.sqrt(2.0 / i), (o, i)).ravel())
            parts.append(rng.normal(1.0, 0.1, o))
            parts.append(rng.normal(0.0, 0.1, o))
        parts.append(rng.normal(0.0, np.sqrt(2.0 / cin), (c3, cin)).ravel())
        parts.append(rng.normal(1.0, 0.1, c3))
        parts.append(rng.normal(0.0, 0.1, c3))
    i = a.channels[-1][2]
    for d in tuple(a.fc_hidden) + (a.n_classes,):
        parts.append(rng.normal(0.0, np.sqrt(2.0 / i), (d, i)).ravel())
        parts.append(rng.normal(0.0, 0.1, d))
        i = d
    blob = np.concatenate(parts).astype(np.float32)
    assert blob.size == weight_count(a)
    return blob
