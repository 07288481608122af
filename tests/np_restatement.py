"""A second, independent, vectorised numpy fp64 restatement of the network (whole network).

Written separately from oracle/oracle.c on purpose: different structure (whole-jet broadcasting, lexsort for the
neighbour order, einsum contractions) so that an indexing or transposition slip in either shows as a mismatch.
Lives under tests/ -- it is a pin for the oracle, not part of it, and not part of the product.
"""
import numpy as np


def split_blob(a, blob):
    blob = np.asarray(blob, np.float64)
    o = 0

    def take(n, shape=None):
        nonlocal o
        v = blob[o:o + n]; o += n
        return v.reshape(shape) if shape else v

    blocks = []
    for l, (c1, c2, c3) in enumerate(a.channels):
        cin = a.block_in(l)
        layers = []
        for (i, w) in ((2 * cin, c1), (c1, c2), (c2, c3)):
            layers.append((take(w * i, (w, i)), take(w), take(w)))
        sc = (take(c3 * cin, (c3, cin)), take(c3), take(c3))
        blocks.append((layers, sc))
    fcs = []
    i = a.channels[-1][2]
    for d in tuple(a.fc_hidden) + (a.n_classes,):
        fcs.append((take(d * i, (d, i)), take(d)))
        i = d
    assert o == blob.size
    return blocks, fcs


def knn_lexsort(s, k):
    """Neighbour lists by full sort of (d, j) pairs; self removed by index."""
    n = s.shape[0]
    diff = s[:, None, :] - s[None, :, :]
    d = np.zeros((n, n))
    for c in range(s.shape[1]):            # index-order accumulation, same association as the definition
        d = d + diff[:, :, c] * diff[:, :, c]
    out = np.full((n, k), -1, np.int64)
    for i in range(n):
        js = np.array([j for j in range(n) if j != i], dtype=np.int64)
        if js.size == 0:
            continue
        order = np.lexsort((js, d[i, js]))
        sel = js[order][:k]
        out[i, :sel.size] = sel
    return out, d


def edgeconv_np(layers, sc, x, nbr):
    n, k = nbr.shape
    valid = nbr >= 0
    xj = x[np.where(valid, nbr, 0)]                      # [n,k,cin]
    xi = np.broadcast_to(x[:, None, :], xj.shape)
    h = np.concatenate([xi, xj - xi], axis=2)
    for (W, s, t) in layers:
        h = np.maximum(np.einsum('nkc,oc->nko', h, W) * s + t, 0.0)
    cnt = valid.sum(1)
    agg = (h * valid[:, :, None]).sum(1) / np.maximum(cnt, 1)[:, None]
    Ws, ss, ts = sc
    return np.maximum(agg + (x @ Ws.T) * ss + ts, 0.0)


def forward_np(a, blob, feats, coords, offsets):
    blocks, fcs = split_blob(a, blob)
    B = len(offsets) - 1
    out = np.zeros((B, a.n_classes))
    for b in range(B):
        s, e = int(offsets[b]), int(offsets[b + 1])
        x = np.asarray(feats[s:e], np.float64)
        p = np.asarray(coords[s:e], np.float64)
        if e > s:
            for l, (layers, sc) in enumerate(blocks):
                nbr, _ = knn_lexsort(p if l == 0 else x, a.k)
                x = edgeconv_np(layers, sc, x, nbr)
            g = x.mean(0)
        else:
            g = np.zeros(a.channels[-1][2])
        z = g
        for i, (W, bias) in enumerate(fcs):
            z = W @ z + bias
            if i < len(fcs) - 1:
                z = np.maximum(z, 0.0)
        out[b] = z
    return out
