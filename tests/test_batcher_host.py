"""Host logic of the dynamic batcher and the load generator, without a GPU: csrc/batcher.cu and csrc/loadgen.cu compiled as
plain C++ with -fsanitize=thread against stand-ins for the CUDA runtime and for gnn_infer_slice
(tests/host/batcher_tsan_main.cpp).  The harness checks that every request receives the logits of its own jets from many
submitting threads and through the closed-loop load generator; ThreadSanitizer must stay silent (race
detection for the mutex / condition-variable batcher)."""
import os
import shutil
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
CSRC = os.path.join(ROOT, "paper_2312_06838_b200", "csrc")


@pytest.mark.skipif(shutil.which("g++") is None, reason="no g++")
def test_batcher_and_loadgen_under_thread_sanitizer(tmp_path):
    exe = str(tmp_path / "batcher_tsan")
    cuda_inc = os.path.join(os.environ.get("CUDA_HOME", "/usr/local/cuda"), "include")
    cmd = ["g++", "-std=c++17", "-O1", "-g", "-fsanitize=thread", "-I" + cuda_inc, "-x", "c++",
           os.path.join(CSRC, "batcher.cu"), os.path.join(CSRC, "loadgen.cu"),
           os.path.join(ROOT, "tests", "host", "batcher_tsan_main.cpp"), "-o", exe, "-pthread"]
    subprocess.run(cmd, check=True, capture_output=True, text=True)
    r = subprocess.run([exe], capture_output=True, text=True, timeout=300,
                       env=dict(os.environ, TSAN_OPTIONS="halt_on_error=0 report_signal_unsafe=0"))
    out = r.stdout + r.stderr
    print(out[-2000:])
    assert "ThreadSanitizer" not in out, "data race reported"
    assert r.returncode == 0 and "wrong results 0" in out
