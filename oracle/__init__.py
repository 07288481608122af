"""TEST INFRASTRUCTURE, NOT THE PRODUCT: ctypes wrapper around oracle/oracle.c (plain fp64 CPU statement of the
hot path; see the header of oracle.c for the passages it follows and the tests that pin it).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this module.
It imports nothing from paper_2312_06838_b200 (the CUDA path) and the CUDA path imports nothing from here.
"""
import ctypes as C
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None

ORC_MAX_BLOCKS, ORC_MAX_FC = 4, 3


class _Arch(C.Structure):
    _fields_ = [("in_features", C.c_int), ("coord_dims", C.c_int), ("k", C.c_int), ("n_blocks", C.c_int),
                ("channels", (C.c_int * 3) * ORC_MAX_BLOCKS), ("n_fc_hidden", C.c_int),
                ("fc_hidden", C.c_int * ORC_MAX_FC), ("n_classes", C.c_int)]


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp, no fast-math (the oracle is timed 'as it stands' by bench.py's cpu_baseline)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_LIB)
        _lib.orc_blob_count.restype = C.c_long
    return _lib


def _arch(a) -> _Arch:
    s = _Arch()
    s.in_features, s.coord_dims, s.k, s.n_blocks = a.in_features, a.coord_dims, a.k, len(a.channels)
    for l, ch in enumerate(a.channels):
        for i in range(3):
            s.channels[l][i] = ch[i]
    s.n_fc_hidden = len(a.fc_hidden)
    for i, d in enumerate(a.fc_hidden):
        s.fc_hidden[i] = d
    s.n_classes = a.n_classes
    return s


def _p(x, t):
    return None if x is None else x.ctypes.data_as(C.POINTER(t))


def max_threads() -> int:
    return int(_load().orc_max_threads())


def blob_count(a) -> int:
    s = _arch(a)
    return int(_load().orc_blob_count(C.byref(s)))


def forward(a, blob, feats, coords, offsets, dumps: bool = False, nthreads: int = 0):
    """Whole forward.  Returns logits [B, n_classes] fp64, or a dict with per-stage dumps when dumps=True:
    nbr [L,N,k] int32 (jet-local, (d,j) order, -1 = none), dk/dk1 [L,N], x (list of [N,C3_l]), g [B,C_last]."""
    lib = _load()
    s = _arch(a)
    blob = np.ascontiguousarray(blob, np.float32)
    assert blob.size == blob_count(a), "weight blob size does not match the architecture"
    feats = np.ascontiguousarray(feats, np.float32).reshape(-1, a.in_features)
    coords = np.ascontiguousarray(coords, np.float32).reshape(-1, a.coord_dims)
    offsets = np.ascontiguousarray(offsets, np.int32)
    B, N, L = offsets.size - 1, int(offsets[-1]), len(a.channels)
    assert feats.shape[0] == N and coords.shape[0] == N
    logits = np.zeros((B, a.n_classes), np.float64)
    nbr = dk = dk1 = xd = g = None
    if dumps:
        nbr = np.full((L, N, a.k), -1, np.int32)
        dk = np.zeros((L, N)); dk1 = np.full((L, N), np.inf)
        xd = np.zeros(N * sum(ch[2] for ch in a.channels))
        g = np.zeros((B, a.channels[-1][2]))
    rc = lib.orc_forward(C.byref(s), _p(blob, C.c_float), _p(feats, C.c_float), _p(coords, C.c_float),
                         _p(offsets, C.c_int), C.c_int(B), _p(logits, C.c_double), _p(nbr, C.c_int),
                         _p(dk, C.c_double), _p(dk1, C.c_double), _p(xd, C.c_double), _p(g, C.c_double),
                         C.c_int(nthreads))
    assert rc == 0
    if not dumps:
        return logits
    xs, o = [], 0
    for ch in a.channels:
        xs.append(xd[o:o + N * ch[2]].reshape(N, ch[2])); o += N * ch[2]
    return {"logits": logits, "nbr": nbr, "dk": dk, "dk1": dk1, "x": xs, "g": g}


def knn(space, offsets, k, nthreads: int = 0):
    """Exact kNN per jet on `space` [N, D] (widened to fp64).  Returns idx [N,k] int32, dk [N], dk1 [N]."""
    lib = _load()
    space = np.ascontiguousarray(space, np.float64)
    offsets = np.ascontiguousarray(offsets, np.int32)
    N, D = space.shape
    idx = np.full((N, k), -1, np.int32); dk = np.zeros(N); dk1 = np.full(N, np.inf)
    lib.orc_knn(_p(space, C.c_double), C.c_int(D), _p(offsets, C.c_int), C.c_int(offsets.size - 1), C.c_int(k),
                _p(idx, C.c_int), _p(dk, C.c_double), _p(dk1, C.c_double), C.c_int(nthreads))
    return idx, dk, dk1


def edgeconv(a, blob, block, x, idx, offsets, nthreads: int = 0):
    """One EdgeConv block given jet-local neighbour indices.  x [N, C_in] -> [N, C3] fp64."""
    lib = _load()
    s = _arch(a)
    blob = np.ascontiguousarray(blob, np.float32)
    x = np.ascontiguousarray(x, np.float64)
    idx = np.ascontiguousarray(idx, np.int32)
    offsets = np.ascontiguousarray(offsets, np.int32)
    assert idx.shape == (x.shape[0], a.k) and x.shape[1] == a.block_in(block)
    y = np.zeros((x.shape[0], a.channels[block][2]))
    lib.orc_edgeconv(C.byref(s), _p(blob, C.c_float), C.c_int(block), _p(x, C.c_double), _p(idx, C.c_int),
                     _p(offsets, C.c_int), C.c_int(offsets.size - 1), _p(y, C.c_double), C.c_int(nthreads))
    return y


def pool_head(a, blob, x, offsets, nthreads: int = 0):
    """Masked global average pool + FC head.  x [N, C_last] -> (logits [B, n_classes], g [B, C_last])."""
    lib = _load()
    s = _arch(a)
    blob = np.ascontiguousarray(blob, np.float32)
    x = np.ascontiguousarray(x, np.float64)
    offsets = np.ascontiguousarray(offsets, np.int32)
    B = offsets.size - 1
    logits = np.zeros((B, a.n_classes)); g = np.zeros((B, a.channels[-1][2]))
    lib.orc_pool_head(C.byref(s), _p(blob, C.c_float), _p(x, C.c_double), _p(offsets, C.c_int), C.c_int(B),
                      _p(logits, C.c_double), _p(g, C.c_double), C.c_int(nthreads))
    return logits, g


def forward_padded(a, blob, feats, coords, mask, nthreads: int = 0):
    """Padded entry (features, coordinates, mask).  R7: masked particles do not exist -- they are
    removed by a stable, order-preserving compaction (mask != 0 keeps a slot) before anything else is computed, so
    whatever sits in a masked slot (NaN, 1e9) is never read."""
    feats = np.asarray(feats, np.float32); coords = np.asarray(coords, np.float32); mask = np.asarray(mask)
    B, P = mask.shape
    keep = mask != 0
    offsets = np.zeros(B + 1, np.int32)
    offsets[1:] = np.cumsum(keep.sum(1))
    f = feats.reshape(B * P, -1)[keep.reshape(-1)]
    c = coords.reshape(B * P, -1)[keep.reshape(-1)]
    return forward(a, blob, f, c, offsets, nthreads=nthreads)


def softmax(logits):
    """Class probabilities from logits [B, n_classes], fp64: p_c = exp(z_c - max z) / sum_c' exp(z_c' - max z) (the textbook
    definition; PAPER.md L262 ends the network in "two nodes", L270 serves their FP32 scores)."""
    z = np.asarray(logits, np.float64)
    e = np.exp(z - z.max(axis=1, keepdims=True))
    return e / e.sum(axis=1, keepdims=True)
