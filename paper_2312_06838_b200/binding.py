"""ctypes binding with the same names as include/gnn.h (gnn_create -> Model, gnn_infer -> Model.infer, ...)."""
import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libgnn.so")
GNN_MAX_BLOCKS, GNN_MAX_FC = 4, 3
FP32_VALIDATION, BF16 = 0, 1
_lib = None


class GnnError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        super().__init__("%s: %s (%d)" % (where, strerror(code), code))


class GnnArch(C.Structure):
    _fields_ = [("in_features", C.c_int32), ("coord_dims", C.c_int32), ("k", C.c_int32), ("n_blocks", C.c_int32),
                ("channels", (C.c_int32 * 3) * GNN_MAX_BLOCKS), ("n_fc_hidden", C.c_int32),
                ("fc_hidden", C.c_int32 * GNN_MAX_FC), ("n_classes", C.c_int32), ("max_particles", C.c_int32),
                ("max_batch_jets", C.c_int32), ("precision", C.c_int32), ("workspace_slices", C.c_int32)]


class BatcherOpts(C.Structure):
    _fields_ = [("max_batch_jets", C.c_int32), ("max_queue_delay_us", C.c_int32), ("n_instances", C.c_int32),
                ("max_pending_requests", C.c_int32)]


class Ticket(C.Structure):
    _fields_ = [("id", C.c_uint64)]


class LoadgenPool(C.Structure):
    _fields_ = [("feats_host", C.c_void_p), ("coords_host", C.c_void_p), ("offsets_host", C.c_void_p),
                ("request_first_jet", C.c_void_p), ("n_requests", C.c_int32), ("in_features", C.c_int32),
                ("coord_dims", C.c_int32), ("n_classes", C.c_int32)]


class LoadgenOpts(C.Structure):
    _fields_ = [("n_clients", C.c_int32), ("warmup_ms", C.c_int32), ("run_ms", C.c_int32)]


class LoadgenResult(C.Structure):
    _fields_ = [("n_requests", C.c_uint64), ("n_jets", C.c_uint64)] + [(k, C.c_double) for k in (
        "seconds", "jets_per_s", "mean_us", "p50_us", "p90_us", "p99_us", "queue_us_mean", "compute_us_mean",
        "mean_batch_jets", "transfer_us_mean", "inference_us_mean")]


def lib():
    """Loads libgnn.so (built in-tree by `python -m paper_2312_06838_b200.build`).  No fallback."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("libgnn.so is not built: run `python -m paper_2312_06838_b200.build` "
                              "(or __graft_entry__.build()); there is no CPU fallback")
        L = C.CDLL(LIB_PATH)
        vp, i32, f32p, i32p = C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p
        L.gnn_weights_bytes.argtypes = [C.POINTER(GnnArch), C.POINTER(C.c_size_t)]
        L.gnn_create.argtypes = [vp, C.c_size_t, C.POINTER(GnnArch), C.c_int, C.POINTER(vp)]
        L.gnn_destroy.argtypes = [vp]; L.gnn_destroy.restype = None
        L.gnn_infer.argtypes = [vp, f32p, f32p, i32p, i32, i32, f32p, vp]
        L.gnn_infer_slice.argtypes = [vp, i32, f32p, f32p, i32p, i32, i32, f32p, vp]
        L.gnn_infer_padded.argtypes = [vp, f32p, f32p, f32p, i32, i32, f32p, vp]
        L.gnn_infer_padded_slice.argtypes = [vp, i32, f32p, f32p, f32p, i32, i32, f32p, vp]
        L.gnn_status_check.argtypes = [vp, i32, vp]
        L.gnn_infer_channel_first.argtypes = [vp, i32, f32p, f32p, f32p, i32, i32, i32, f32p, vp]
        L.gnn_softmax.argtypes = [f32p, i32, i32, f32p, vp]
        L.gnn_infer_host.argtypes = [vp, i32, vp, vp, vp, i32, i32, vp, vp]
        L.gnn_infer_host_begin.argtypes = [vp, i32, vp, vp, vp, i32, i32, vp, vp]
        L.gnn_infer_host_end.argtypes = [vp, i32, vp]
        L.gnn_profile_enable.argtypes = [vp, i32, i32]
        L.gnn_profile_read.argtypes = [vp, i32, i32, C.POINTER(C.c_float), C.POINTER(i32), C.POINTER(i32)]
        L.gnn_profile_stage_name.argtypes = [vp, i32, i32]; L.gnn_profile_stage_name.restype = C.c_char_p
        L.gnn_strerror.argtypes = [C.c_int]; L.gnn_strerror.restype = C.c_char_p
        L.gnn_launch_count.argtypes = [vp]; L.gnn_launch_count.restype = C.c_int64
        L.gnn_debug_knn.argtypes = [vp, f32p, i32, i32p, i32, i32, i32, i32p, vp]
        L.gnn_knn_noalloc.argtypes = [f32p, i32, i32p, i32, i32, i32, i32, i32p, vp]
        L.gnn_debug_edgeconv.argtypes = [vp, i32, f32p, i32p, i32p, i32, i32, f32p, vp]
        L.gnn_debug_pool_head.argtypes = [vp, f32p, i32p, i32, i32, f32p, vp]
        L.gnn_debug_edgeconv_pool.argtypes = [vp, f32p, i32p, i32p, i32, i32, f32p, vp]
        L.gnn_batcher_create.argtypes = [vp, C.POINTER(BatcherOpts), C.POINTER(vp)]
        L.gnn_batcher_submit.argtypes = [vp, vp, vp, vp, i32, vp, C.POINTER(Ticket)]
        L.gnn_batcher_wait.argtypes = [vp, Ticket, C.c_int64, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.gnn_batcher_wait_ex.argtypes = [vp, Ticket, C.c_int64, C.c_void_p]
        L.gnn_batcher_stats.argtypes = [vp, C.POINTER(C.c_uint64), C.POINTER(C.c_uint64), C.POINTER(C.c_uint64),
                                        C.POINTER(C.c_double)]
        L.gnn_batcher_destroy.argtypes = [vp]; L.gnn_batcher_destroy.restype = None
        L.gnn_bdt_create.argtypes = [vp, vp, vp, i32, i32, i32, C.c_int, C.POINTER(vp)]
        L.gnn_bdt_destroy.argtypes = [vp]; L.gnn_bdt_destroy.restype = None
        L.gnn_bdt_infer.argtypes = [vp, f32p, C.c_int64, f32p, vp]
        L.gnn_bdt_infer_host.argtypes = [vp, vp, C.c_int64, vp, vp]
        L.gnn_loadgen_run.argtypes = [vp, C.POINTER(LoadgenPool), C.POINTER(LoadgenOpts), C.POINTER(LoadgenResult)]
        _lib = L
    return _lib


def strerror(code: int) -> str:
    return lib().gnn_strerror(int(code)).decode()


def arch_struct(a, max_batch_jets=1024, precision=FP32_VALIDATION, workspace_slices=1, max_particles=None) -> GnnArch:
    """Builds a gnn_arch from any object with the fields of synth.Arch (plain data; nothing is imported)."""
    s = GnnArch()
    s.in_features, s.coord_dims, s.k, s.n_blocks = a.in_features, a.coord_dims, a.k, len(a.channels)
    for l, ch in enumerate(a.channels):
        for i in range(3):
            s.channels[l][i] = ch[i]
    s.n_fc_hidden = len(a.fc_hidden)
    for i, d in enumerate(a.fc_hidden):
        s.fc_hidden[i] = d
    s.n_classes = a.n_classes
    s.max_particles = max_particles or a.max_particles
    s.max_batch_jets, s.precision, s.workspace_slices = max_batch_jets, precision, workspace_slices
    return s


def weights_bytes(arch: GnnArch) -> int:
    n = C.c_size_t(0)
    rc = lib().gnn_weights_bytes(C.byref(arch), C.byref(n))
    if rc != 0:
        raise GnnError(rc, "gnn_weights_bytes")
    return int(n.value)


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _hptr(t):
    if t is None:
        return None
    if isinstance(t, np.ndarray):
        return t.ctypes.data_as(C.c_void_p)
    return C.c_void_p(t.data_ptr())


def _stream(stream):
    import torch
    s = stream if stream is not None else torch.cuda.current_stream()
    return C.c_void_p(s.cuda_stream)


def knn_noalloc(space, offsets, k, max_particles=128, idx=None, stream=None):
    """gnn_knn_noalloc: exact kNN with no gnn_model and no device allocation inside the library (its scratch is a fixed
    array inside libgnn.so; at most 1024 jets / 8192 particles per call; calls must not overlap on the GPU).  Pass `idx`
    ([N, k] int32, device) to keep this wrapper from allocating too; torch tensors on the current device."""
    import torch
    N, D = space.shape
    if idx is None:
        idx = torch.full((N, k), -7, dtype=torch.int32, device=space.device)
    rc = lib().gnn_knn_noalloc(_ptr(space), D, _ptr(offsets), offsets.numel() - 1, N, max_particles, k, _ptr(idx),
                               _stream(stream))
    if rc != 0:
        raise GnnError(rc, "gnn_knn_noalloc")
    return idx


class Model:
    """gnn_model.  Tensors passed to infer* are torch CUDA tensors (fp32 / int32, contiguous)."""

    def __init__(self, arch: GnnArch, weights: np.ndarray, device: int = 0):
        w = np.ascontiguousarray(weights, dtype=np.float32)
        h = C.c_void_p()
        rc = lib().gnn_create(w.ctypes.data_as(C.c_void_p), w.nbytes, C.byref(arch), device, C.byref(h))
        if rc != 0:
            raise GnnError(rc, "gnn_create")
        self.h, self.arch, self.device = h, arch, device

    def close(self):
        if getattr(self, "h", None):
            lib().gnn_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc, where):
        if rc != 0:
            raise GnnError(rc, where)

    def infer(self, feats, coords, offsets, logits=None, stream=None, slice=0):
        import torch
        B, N = offsets.numel() - 1, feats.shape[0]
        if logits is None:
            logits = torch.empty((B, self.arch.n_classes), dtype=torch.float32, device=feats.device)
        self._check(lib().gnn_infer_slice(self.h, slice, _ptr(feats), _ptr(coords), _ptr(offsets), B, N, _ptr(logits),
                                          _stream(stream)), "gnn_infer")
        return logits

    def infer_padded(self, feats, coords, mask, logits=None, stream=None, slice=0):
        import torch
        B, P = mask.shape
        if logits is None:
            logits = torch.empty((B, self.arch.n_classes), dtype=torch.float32, device=mask.device)
        self._check(lib().gnn_infer_padded_slice(self.h, slice, _ptr(feats), _ptr(coords), _ptr(mask), B, P, _ptr(logits),
                                                 _stream(stream)), "gnn_infer_padded")
        return logits

    def infer_channel_first(self, points, features, mask, softmax=False, out=None, stream=None, slice=0):
        """gnn_infer_channel_first: points [B, CD, P], features [B, F, P], mask [B, 1, P] device tensors."""
        import torch
        B, P = int(features.shape[0]), int(features.shape[2])
        if out is None:
            out = torch.empty((B, self.arch.n_classes), dtype=torch.float32, device=features.device)
        self._check(lib().gnn_infer_channel_first(self.h, slice, _ptr(points), _ptr(features), _ptr(mask), B, P, int(bool(softmax)),
                                                  _ptr(out), _stream(stream)), "gnn_infer_channel_first")
        return out

    def infer_host(self, feats, coords, offsets, logits, stream=None, slice=0):
        """gnn_infer_host: host tensors / arrays in (torch CPU tensors, ideally pinned, or numpy), logits written into
        `logits` (host).  Blocks until the logits are in host memory."""
        B, N = int(offsets.shape[0]) - 1, int(feats.shape[0])
        self._check(lib().gnn_infer_host(self.h, slice, _hptr(feats), _hptr(coords), _hptr(offsets), B, N,
                                         _hptr(logits), _stream(stream)), "gnn_infer_host")
        return logits

    def infer_host_begin(self, feats, coords, offsets, logits, stream=None, slice=0):
        """gnn_infer_host_begin: enqueue copies + forward on `stream`; gnn_infer_host_end(slice) collects (pinned host tensors)."""
        B, N = int(offsets.shape[0]) - 1, int(feats.shape[0])
        self._check(lib().gnn_infer_host_begin(self.h, slice, _hptr(feats), _hptr(coords), _hptr(offsets), B, N,
                                               _hptr(logits), _stream(stream)), "gnn_infer_host_begin")

    def infer_host_end(self, stream=None, slice=0):
        self._check(lib().gnn_infer_host_end(self.h, slice, _stream(stream)), "gnn_infer_host_end")

    def profile_enable(self, on=True, slice=0):
        self._check(lib().gnn_profile_enable(self.h, slice, 1 if on else 0), "gnn_profile_enable")

    def profile_read(self, slice=0):
        """-> (list of (stage name, mean ms), forwards averaged)"""
        ms = (C.c_float * 64)()
        ns, nf = C.c_int32(0), C.c_int32(0)
        self._check(lib().gnn_profile_read(self.h, slice, 64, ms, C.byref(ns), C.byref(nf)), "gnn_profile_read")
        names = [(lib().gnn_profile_stage_name(self.h, slice, i) or b"?").decode() for i in range(ns.value)]
        return list(zip(names, [float(ms[i]) for i in range(ns.value)])), int(nf.value)

    def status_check(self, slice=0, stream=None) -> int:
        return int(lib().gnn_status_check(self.h, slice, _stream(stream)))

    def launch_count(self) -> int:
        return int(lib().gnn_launch_count(self.h))

    def debug_knn(self, space, offsets, k, stream=None):
        import torch
        N, D = space.shape
        idx = torch.full((N, k), -7, dtype=torch.int32, device=space.device)
        self._check(lib().gnn_debug_knn(self.h, _ptr(space), D, _ptr(offsets), offsets.numel() - 1, N, k, _ptr(idx),
                                        _stream(stream)), "gnn_debug_knn")
        return idx

    def debug_edgeconv(self, block, x, idx, offsets, stream=None):
        import torch
        N = x.shape[0]
        y = torch.empty((N, self.arch.channels[block][2]), dtype=torch.float32, device=x.device)
        self._check(lib().gnn_debug_edgeconv(self.h, block, _ptr(x), _ptr(idx), _ptr(offsets), offsets.numel() - 1, N,
                                             _ptr(y), _stream(stream)), "gnn_debug_edgeconv")
        return y

    def debug_edgeconv_pool(self, x, idx, offsets, stream=None):
        import torch
        B = offsets.numel() - 1
        C_last = self.arch.channels[self.arch.n_blocks - 1][2]
        g = torch.empty((B, C_last), dtype=torch.float32, device=x.device)
        self._check(lib().gnn_debug_edgeconv_pool(self.h, _ptr(x), _ptr(idx), _ptr(offsets), B, x.shape[0], _ptr(g),
                                                  _stream(stream)), "gnn_debug_edgeconv_pool")
        return g

    def debug_pool_head(self, x, offsets, stream=None):
        import torch
        B = offsets.numel() - 1
        logits = torch.empty((B, self.arch.n_classes), dtype=torch.float32, device=x.device)
        self._check(lib().gnn_debug_pool_head(self.h, _ptr(x), _ptr(offsets), B, x.shape[0], _ptr(logits),
                                              _stream(stream)), "gnn_debug_pool_head")
        return logits


class Batcher:
    """gnn_batcher: host dynamic batcher.  submit() takes numpy host arrays; wait() fills the logits array."""

    def __init__(self, model: Model, max_batch_jets=1024, max_queue_delay_us=1000, n_instances=2,
                 max_pending_requests=0):
        self.model = model
        o = BatcherOpts(max_batch_jets, max_queue_delay_us, n_instances, max_pending_requests)
        h = C.c_void_p()
        rc = lib().gnn_batcher_create(model.h, C.byref(o), C.byref(h))
        if rc != 0:
            raise GnnError(rc, "gnn_batcher_create")
        self.h = h
        self.n_classes = model.arch.n_classes

    def submit(self, feats: np.ndarray, coords: np.ndarray, offsets: np.ndarray, logits_out: np.ndarray = None):
        n_jets = offsets.size - 1
        if logits_out is None:
            logits_out = np.empty((n_jets, self.n_classes), np.float32)
        t = Ticket()
        rc = lib().gnn_batcher_submit(self.h, feats.ctypes.data_as(C.c_void_p), coords.ctypes.data_as(C.c_void_p),
                                      offsets.ctypes.data_as(C.c_void_p), n_jets,
                                      logits_out.ctypes.data_as(C.c_void_p), C.byref(t))
        if rc != 0:
            raise GnnError(rc, "gnn_batcher_submit")
        return t, logits_out

    def wait(self, ticket, timeout_us=-1):
        q, c = C.c_double(0), C.c_double(0)
        rc = lib().gnn_batcher_wait(self.h, ticket, timeout_us, C.byref(q), C.byref(c))
        return int(rc), q.value, c.value

    def wait_ex(self, ticket, timeout_us=-1):
        """gnn_batcher_wait_ex -> (status, {queue_us, compute_us, transfer_us, inference_us})"""
        t = (C.c_double * 4)()
        rc = lib().gnn_batcher_wait_ex(self.h, ticket, timeout_us, C.cast(t, C.c_void_p))
        return int(rc), dict(zip(("queue_us", "compute_us", "transfer_us", "inference_us"), list(t)))

    def stats(self):
        a, b, c, d = C.c_uint64(0), C.c_uint64(0), C.c_uint64(0), C.c_double(0)
        lib().gnn_batcher_stats(self.h, C.byref(a), C.byref(b), C.byref(c), C.byref(d))
        return {"n_requests": a.value, "n_jets": b.value, "n_launches": c.value, "mean_batch_jets": d.value}

    def loadgen(self, feats: np.ndarray, coords: np.ndarray, offsets: np.ndarray, request_first_jet: np.ndarray,
                n_clients: int, warmup_ms: int = 500, run_ms: int = 2000) -> dict:
        """gnn_loadgen_run: closed-loop native client threads over a pool of requests cut from one ragged host batch."""
        feats = np.ascontiguousarray(feats, np.float32); coords = np.ascontiguousarray(coords, np.float32)
        offsets = np.ascontiguousarray(offsets, np.int32); rfj = np.ascontiguousarray(request_first_jet, np.int32)
        a = self.model.arch
        pool = LoadgenPool(feats.ctypes.data, coords.ctypes.data, offsets.ctypes.data, rfj.ctypes.data, rfj.size - 1,
                           a.in_features, a.coord_dims, a.n_classes)
        o = LoadgenOpts(n_clients, warmup_ms, run_ms)
        r = LoadgenResult()
        rc = lib().gnn_loadgen_run(self.h, C.byref(pool), C.byref(o), C.byref(r))
        if rc != 0:
            raise GnnError(rc, "gnn_loadgen_run")
        return {k: getattr(r, k) for k, _ in LoadgenResult._fields_}

    def close(self):
        if getattr(self, "h", None):
            lib().gnn_batcher_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class Bdt:
    """gnn_bdt: boosted-decision-tree inference (include/gnn.h).  Marshalling only."""

    def __init__(self, feature: np.ndarray, threshold: np.ndarray, leaf: np.ndarray, n_features: int, device: int = 0):
        feature = np.ascontiguousarray(feature, np.int32); threshold = np.ascontiguousarray(threshold, np.float32)
        leaf = np.ascontiguousarray(leaf, np.float32)
        n_trees, n_int = feature.shape
        depth = int(n_int + 1).bit_length() - 1
        self.n_features = int(n_features)
        h = C.c_void_p()
        rc = lib().gnn_bdt_create(feature.ctypes.data, threshold.ctypes.data, leaf.ctypes.data, n_trees, depth, self.n_features,
                                  device, C.byref(h))
        if rc != 0:
            raise GnnError(rc, "gnn_bdt_create")
        self.h = h

    def infer(self, x, out=None, stream=None):
        import torch
        N = int(x.shape[0])
        if out is None:
            out = torch.empty((N, 2), dtype=torch.float32, device=x.device)
        rc = lib().gnn_bdt_infer(self.h, _ptr(x), N, _ptr(out), _stream(stream))
        if rc != 0:
            raise GnnError(rc, "gnn_bdt_infer")
        return out

    def infer_host(self, x, out, stream=None):
        rc = lib().gnn_bdt_infer_host(self.h, _hptr(x), int(x.shape[0]), _hptr(out), _stream(stream))
        if rc != 0:
            raise GnnError(rc, "gnn_bdt_infer_host")
        return out

    def close(self):
        if getattr(self, "h", None):
            lib().gnn_bdt_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
