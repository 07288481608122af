"""Host-side checks that need no GPU: libgnn.so builds, loads and exports every symbol include/gnn.h declares;
argument validation that happens before any CUDA call."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2312_06838_b200 import build
    build.build()
    import paper_2312_06838_b200 as gnn
    return gnn.lib()


def test_exports_every_declared_symbol(lib):
    hdr = open(os.path.join(ROOT, "include", "gnn.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    names = sorted(set(re.findall(r"\b(gnn_[a-z_0-9]+)\s*\(", hdr)))
    assert len(names) == 34
    for n in names:
        assert hasattr(lib, n), "libgnn.so does not export %s" % n


def test_weights_bytes_and_arch_validation(lib):
    import paper_2312_06838_b200 as gnn
    for name, cnt in (("particlenet", 366146), ("wide", 1453186), ("tiny", 2754)):
        a = gnn.arch_struct(synth.ARCHS[name])
        assert gnn.weights_bytes(a) == 4 * cnt == 4 * synth.weight_count(synth.ARCHS[name])
    bad = gnn.arch_struct(synth.ARCHS["particlenet"])
    bad.k = 0
    n = C.c_size_t(0)
    assert lib.gnn_weights_bytes(C.byref(bad), C.byref(n)) == -2
    bad = gnn.arch_struct(synth.ARCHS["particlenet"])
    bad.channels[1][1] = 100                       # not a multiple of 8
    assert lib.gnn_weights_bytes(C.byref(bad), C.byref(n)) == -2
    assert lib.gnn_weights_bytes(None, C.byref(n)) == -1
    assert b"no CPU fallback" in lib.gnn_strerror(-5)


def test_create_rejects_wrong_blob_size_before_touching_cuda(lib):
    import paper_2312_06838_b200 as gnn
    a = gnn.arch_struct(synth.ARCHS["tiny"])
    w = np.zeros(10, np.float32)
    h = C.c_void_p()
    assert lib.gnn_create(w.ctypes.data_as(C.c_void_p), w.nbytes, C.byref(a), 0, C.byref(h)) == -3
    assert lib.gnn_create(None, 0, C.byref(a), 0, C.byref(h)) == -1


def test_no_cpu_fallback_without_a_gpu(lib):
    """On a box without a CUDA device gnn_create must fail loudly (GNN_ERR_CUDA), never compute on the CPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    import paper_2312_06838_b200 as gnn
    a = synth.ARCHS["tiny"]
    with pytest.raises(gnn.GnnError) as e:
        gnn.Model(gnn.arch_struct(a), synth.make_weights(a))
    assert e.value.code == -5


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2312_06838_b200")
    for dp, _, fs in os.walk(pkg):
        if os.path.basename(dp) == "build":
            continue
        for f in fs:
            if f.endswith((".py", ".cu", ".h", ".cpp", ".cuh")):
                src = open(os.path.join(dp, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle", src, flags=re.M), f
                assert "oracle/" not in src and "liboracle" not in src, f
    osrc = open(os.path.join(ROOT, "oracle", "__init__.py")).read() + open(os.path.join(ROOT, "oracle", "oracle.c")).read()
    assert not re.search(r"^\s*(import|from)\s+paper_2312_06838_b200", osrc, flags=re.M)
    assert "gnn.h\"" not in osrc


def test_noalloc_entry_allocates_nothing_and_its_scratch_is_the_documented_size():
    """gnn_knn_noalloc is the entry for callers that may not allocate device memory: its source (and the helper that looks up the
    scratch address) must not name an allocating call, the scratch must be a file-scope static __device__ array aligned to 256
    bytes, and its size must be what gnn.h and the README tell those callers (about 4.1 MiB, 1024 jets / 8192 particles)."""
    src = open(os.path.join(ROOT, "paper_2312_06838_b200", "csrc", "knn.cu")).read()
    tail = src[src.index("constexpr int NOALLOC_MAX_JETS"):]
    code = re.sub(r"//[^\n]*", "", tail)                                 # comments may (and do) name cudaMalloc
    for banned in ("cudaMalloc", "cudaFree", "cudaHostAlloc", "cudaMallocAsync", "new ", "std::vector"):
        assert banned not in code, banned
    assert "cudaGetSymbolAddress" in code and "static __device__ __align__(256) unsigned char knn_noalloc_scratch" in code
    jets = int(re.search(r"NOALLOC_MAX_JETS = (\d+)", tail).group(1))
    rows = int(re.search(r"NOALLOC_MAX_ROWS = (\d+)", tail).group(1))
    assert (jets, rows) == (1024, 8192)
    size = 256 + 2 * 4 * jets + 8 * rows + 4 * rows * 128                # status/meta | jet_start | jet_n | pjet | dm
    assert size == 4268288 and abs(size / 2 ** 20 - 4.1) < 0.05
    hdr = open(os.path.join(ROOT, "include", "gnn.h")).read()
    assert "B <= 1024 jets and N <= 8192 particles" in hdr and "4.1 MiB" in hdr
    assert "4.1 MiB" in open(os.path.join(ROOT, "README.md")).read()
