"""ThreadSanitizer pass over the host side of the library (many clients, one
server): pp_api.cpp, pp_ipc.cpp and pp_multi.cpp are compiled with -fsanitize=thread against a fake CUDA runtime and
fake kernels (tests/tsan/) and driven from many threads.  A data race, a failed check or a hang fails the test."""
import os
import shutil
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.skipif(shutil.which("g++") is None, reason="needs g++ with -fsanitize=thread")
def test_host_side_is_race_free_under_tsan(tmp_path):
    r = subprocess.run([os.path.join(ROOT, "tests", "tsan", "build_and_run.sh"), str(tmp_path)], capture_output=True,
                       text=True, timeout=600)
    assert "ThreadSanitizer" not in r.stderr, r.stderr[-4000:]
    assert r.returncode == 0 and r.stdout.strip().endswith("OK"), (r.returncode, r.stdout[-2000:], r.stderr[-2000:])
    assert "relaunches" in r.stdout and "ipc over 2 devices" in r.stdout
