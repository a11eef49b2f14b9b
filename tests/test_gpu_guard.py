"""-m gpu: the guard build of the library (tests/libpp_guard.so, -DPP_GUARD) in place of compute-sanitizer's memcheck,
which the pool's wrapper refuses (PAPER.md:47 is about staying inside a memory limit).

In that build every piece of the device workspace (source records, prefix sums, tile table, both resume lists, Status +
hit ring, resident batch) is followed by a 256-byte zone of a known pattern that the host reads back after EVERY launch,
and the propagation kernel checks its own index arithmetic (source index, tile table entries, photon index, fate index)
and reports a code instead of storing out of bounds.  The scenarios are the ones that stress the bounded buffers: a hit
ring far too small (hundreds of relaunches through the resume lists), launches that start inside a source, the fate
dump, C0 and a slice of C1.  They run in a process of their own (the library is chosen when the binding is first
loaded: environment variable PP_LIB); the hits must equal those of the product build bit for bit."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

from paper_2405_05700_b200 import binding as B
from paper_2405_05700_b200 import workloads as W

from gpu_util import gpu_run, gpu_run_resident

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def scenarios():
    """(name, runner) pairs; a runner returns a structured array that must not depend on the build."""
    geo, ice = W.geometry_full(radius=1.5), W.ice_layered()
    c2 = W.sources_c2(seed=5, n_events=40)
    c2.src[:, 7] *= 3.0
    few = W.sources_c1().subset(slice(0, 6))
    few.src[:, 7] = np.array([0.9993, 5.0, 0.0031, 2.0, 0.0007, 1.5], np.float32)
    c1 = W.sources_c1().subset(slice(0, 60))
    c1.src[:, 7] = 0.3
    return [
        ("tiny hit ring: relaunches through the resume lists",
         lambda: gpu_run(geo, ice, c2, 9, hit_ring_bytes=2 * 32 * 64, launch_photons_target=10 ** 6)[0]),
        ("launches that start inside a source", lambda: gpu_run(W.geometry_full(radius=2.0), ice, few, 4, launch_photons_target=10000)[0]),
        ("C0 with the fate dump", lambda: gpu_run_resident(W.geometry_single_string(radius=1.0), W.ice_homogeneous(),
                                                            W.sources_c0(seed=1, n_photons=2.0e5, toward_string=True), 1,
                                                            want_fates=True)[1]),
        ("C1 slice with the fate dump, real radius", lambda: gpu_run_resident(W.geometry_full(), ice, c1, 0, want_fates=True)[1]),
        ("C1 slice through the server, several launches", lambda: gpu_run(W.geometry_full(radius=1.0), ice, c1, 0, launch_photons_target=50000)[0]),
    ]


def _child(out_dir):
    L = B.load_library()
    import ctypes as C
    L.pp_guard_zone_checks.restype = C.c_uint64  # exported by the guard build only
    info = {"lib": B.LIB_PATH, "scenarios": []}
    for i, (name, run) in enumerate(scenarios()):
        before = int(L.pp_guard_zone_checks())
        launches0 = B.kernel_launch_count()
        a = run()
        np.save(os.path.join(out_dir, f"s{i}.npy"), a)
        info["scenarios"].append({"name": name, "records": int(len(a)), "zone_checks": int(L.pp_guard_zone_checks()) - before,
                                  "kernel_launches": B.kernel_launch_count() - launches0})
    print("GUARD_INFO " + json.dumps(info))


def test_guard_build_finds_nothing_and_agrees_with_the_product_build(tmp_path):
    from conftest import GUARD_LIB, build_guard_library
    build_guard_library()
    env = dict(os.environ, PP_LIB=GUARD_LIB, PYTHONPATH=os.pathsep.join([ROOT, os.path.join(ROOT, "tests")]))
    r = subprocess.run([sys.executable, "-c", f"import test_gpu_guard as T; T._child({str(tmp_path)!r})"],
                       env=env, capture_output=True, text=True, timeout=800)
    assert r.returncode == 0, r.stdout[-3000:] + r.stderr[-3000:]   # a tripped guard surfaces as PP_E_CUDA "internal: guard ..."
    info = json.loads([ln for ln in r.stdout.splitlines() if ln.startswith("GUARD_INFO ")][-1][len("GUARD_INFO "):])
    assert info["lib"].endswith("libpp_guard.so")
    for i, (name, run) in enumerate(scenarios()):
        sc = info["scenarios"][i]
        assert sc["zone_checks"] > 0 and sc["kernel_launches"] > 0, sc     # the checks really ran
        assert np.array_equal(np.load(os.path.join(str(tmp_path), f"s{i}.npy")), run()), name
    assert info["scenarios"][0]["kernel_launches"] > 100                    # the resume lists were exercised
    try:
        os.makedirs("gpurun_out", exist_ok=True)
        with open(os.path.join("gpurun_out", "r03_guard.json"), "w") as f:
            json.dump(info, f, indent=1)
    except OSError:
        pass
