"""CPU tests of the library's host logic: the shared library loads and exports every symbol that
include/pp.h declares; input validation; photon counting; launch cutting (a1); replica reduction
(world_size 2, gloo).  No compute call touches a GPU here."""
import os
import re
import subprocess
import sys

import numpy as np
import pytest

from paper_2405_05700_b200 import binding as B
from paper_2405_05700_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "pp.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(pp_[a-z_]+)\s*\(", hdr))
    assert {"pp_create", "pp_submit", "pp_collect", "pp_flush", "pp_run_resident"} <= declared
    lib = B.load_library()
    for name in declared:
        assert hasattr(lib, name), name
    assert declared == set(B.EXPORTS)
    assert b"sm_100a" in lib.pp_version()


def test_library_holds_sm100a_code():
    out = subprocess.run(["cuobjdump", "-lelf", B.LIB_PATH], capture_output=True, text=True)
    if out.returncode != 0:
        pytest.skip("cuobjdump not available")
    assert "sm_100a" in out.stdout


def test_record_layouts_match_the_header():
    assert B.SOURCE_DTYPE.itemsize == 32 and B.HIT_DTYPE.itemsize == 32 and B.FATE_DTYPE.itemsize == 40
    assert B.HIT_DTYPE.fields["time_ns"][1] == 16 and B.FATE_DTYPE.fields["time_ns"][1] == 16


def test_check_inputs_accepts_the_configs():
    assert B.check_inputs(W.geometry_single_string(), W.ice_homogeneous()) == 0
    assert B.check_inputs(W.geometry_full(), W.ice_layered()) == 0


def test_check_inputs_rejects_bad_values():
    geo, ice = W.geometry_full(), W.ice_layered()
    bad = W.ice_layered(); bad.abs_len[3] = 0.0
    assert B.check_inputs(geo, bad) == -1
    bad = W.ice_layered(); bad.scat_len[7] = np.nan
    assert B.check_inputs(geo, bad) == -1
    bad = W.ice_layered(); bad.g = 1.0
    assert B.check_inputs(geo, bad) == -1
    bad = W.ice_layered(); bad.dz = 0.0
    assert B.check_inputs(geo, bad) == -1
    bad = W.ice_layered(); bad.cos_cherenkov = 1.5
    assert B.check_inputs(geo, bad) == -1
    g2 = W.geometry_full(); g2.radius = -1.0
    assert B.check_inputs(g2, ice) == -1
    g2 = W.geometry_full(); g2.xyz[5, 1] = np.inf
    assert B.check_inputs(g2, ice) == -1


def test_unsupported_geometry_needs_the_brute_force_flag():
    ice = W.ice_layered()
    g = W.geometry_single_string()
    g.xyz[10, 2] += 3.0  # breaks the uniform pitch of the line
    assert B.check_inputs(g, ice) == -6
    assert B.check_inputs(g, ice, B.FLAG_BRUTE_FORCE_DOMS) == 0
    rng = np.random.default_rng(0)
    cloud = W.Geometry(xyz=rng.uniform(-500, 500, size=(700, 3)).astype(np.float32))  # 700 one-DOM lines
    assert B.check_inputs(cloud, ice) == -6
    few = W.Geometry(xyz=rng.uniform(-500, 500, size=(40, 3)).astype(np.float32))  # arbitrary points = 40 lines of 1
    assert B.check_inputs(few, ice) == 0


def test_photon_count():
    assert B.photon_count(10.0) == 100000
    assert B.photon_count(0.0) == 0
    assert B.photon_count(0.00016) == 2
    assert B.photon_count(4.0e5) == 4 * 10 ** 9
    with pytest.raises(B.PPError) as e:
        B.photon_count(5.0e5)  # 5e9 >= 2^32
    assert e.value.code == -4
    with pytest.raises(B.PPError):
        B.photon_count(-1.0)


def _check_plan(counts, target):
    plan = B.plan_launches(counts, target)
    counts = np.asarray(counts, dtype=np.uint64)
    covered = np.zeros(len(counts), dtype=np.uint64)
    prev_end_src, prev_end_off = 0, 0
    for k, (first, n, g0, g1) in enumerate(plan):
        assert n >= 1 and g1 > g0
        assert g1 - g0 <= target
        if k + 1 < len(plan):
            assert g1 - g0 == target  # only the last launch of a flush may be short
        cum = np.concatenate([[0], np.cumsum(counts[first:first + n])])
        assert g0 < cum[1] or counts[first] == 0 or n == 1 or g0 <= cum[1]
        assert g1 <= cum[-1]
        # continuity: this launch starts where the previous one stopped
        assert first == prev_end_src or (first > prev_end_src and np.all(counts[prev_end_src + (1 if prev_end_off else 0):first] == 0)
                                         and (prev_end_off == 0 or prev_end_off == counts[prev_end_src]))
        for i in range(n):
            lo, hi = max(int(cum[i]), g0), min(int(cum[i + 1]), g1)
            if hi > lo:
                assert covered[first + i] == lo - int(cum[i])  # photon ranges of a source are consecutive
                covered[first + i] += hi - lo
        last = first + n - 1
        prev_end_src, prev_end_off = last, int(covered[last])
        if covered[last] == counts[last]:
            prev_end_src, prev_end_off = last + 1, 0
    assert np.array_equal(covered, counts)  # every photon exactly once
    return plan


def test_launch_cutting_small_cases():
    assert B.plan_launches([], 10) == []
    assert B.plan_launches([0, 0, 0], 10) == []
    assert _check_plan([5], 10) == [(0, 1, 0, 5)]
    assert _check_plan([25], 10) == [(0, 1, 0, 10), (0, 1, 10, 20), (0, 1, 20, 25)]
    assert _check_plan([5, 0, 10, 3, 100, 1], 8)[0] == (0, 3, 0, 8)
    _check_plan([10, 10, 10], 10)
    _check_plan([1] * 37, 5)
    _check_plan([0, 7, 0, 0, 9, 0], 4)


def test_launch_cutting_heavy_tailed_random():
    rng = np.random.default_rng(1)
    for trial in range(20):
        n = int(rng.integers(1, 400))
        counts = np.floor(np.exp(rng.uniform(0, 12, size=n)) * (rng.uniform(size=n) < 0.8)).astype(np.uint32)
        target = int(rng.integers(1, 50000))
        _check_plan(counts, target)


def test_launch_cutting_config_c2_shape():
    s = W.sources_c2()
    counts = np.array([B.photon_count(e) for e in s.src[:, 7]], dtype=np.uint32)
    plan = _check_plan(counts, 10 ** 8)
    assert len(plan) == 2 and int(counts.sum()) > 10 ** 8


GLOO_SCRIPT = r"""
import os, sys
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
from paper_2405_05700_b200 import replicas
dist.init_process_group("gloo")
r = dist.get_rank()
tmax, wsum = replicas.reduce_results(dist, torch.device("cpu"), {{"a": 1.0 + r, "b": 5.0 - r}}, {{"photons": 100.0 * (r + 1)}})
assert tmax == {{"a": 2.0, "b": 5.0}}, tmax
assert wsum == {{"photons": 300.0}}, wsum
assert replicas.aggregate_throughput(dist, torch.device("cpu"), 100.0 * (r + 1), 2.0 + r) == 300.0 / 3.0
assert replicas.replica_seed(7, r) == 7 + r
dist.destroy_process_group()
open(os.path.join({out!r}, "ok%d" % r), "w").write("ok")
"""


def test_replica_reduction_world_size_2_gloo(tmp_path):
    script = tmp_path / "gloo_replicas.py"
    script.write_text(GLOO_SCRIPT.format(root=ROOT, out=str(tmp_path)))
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
           "--master-port", "29571", str(script)]
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=240)
    assert out.returncode == 0, out.stdout + out.stderr
    assert (tmp_path / "ok0").exists() and (tmp_path / "ok1").exists()


def test_replica_reduction_single_process():
    from paper_2405_05700_b200 import replicas
    t, w = replicas.reduce_results(None, None, {"x": 3.0}, {"y": 4.0})
    assert t == {"x": 3.0} and w == {"y": 4.0}


def test_roofline_constant_goes_stale_when_a_kernel_source_changes(tmp_path, monkeypatch):
    """bench.py trusts profiles/instr_per_flight.json only for the exact kernel sources + nvcc flags it was measured
    on (SHA-256): touching a comment in pp_kernels.cu without re-measuring must drop the roofline."""
    import json
    import shutil
    import sys
    sys.path.insert(0, ROOT) if ROOT not in sys.path else None
    import bench
    from paper_2405_05700_b200 import build as pp_build
    csrc = tmp_path / "csrc"
    csrc.mkdir()
    for name in bench.KERNEL_SOURCES:
        shutil.copy(os.path.join(pp_build.CSRC, name), csrc / name)
    monkeypatch.setattr(pp_build, "CSRC", str(csrc))
    monkeypatch.delenv("PP_NVCC_EXTRA", raising=False)
    f = tmp_path / "instr_per_flight.json"
    monkeypatch.setattr(bench, "INSTR_PER_FLIGHT_FILE", str(f))
    f.write_text(json.dumps({"thread_instructions_per_flight": 321.0, "dram_bytes_per_launch": 1.0e6,
                             "fp32_flops_per_flight": 150.0, "kernel_sources_sha256": bench.kernel_source_hash()}))
    ipf, dram, note, fpf = bench.load_instr_per_flight()
    assert ipf == 321.0 and dram == 1.0e6 and fpf == 150.0
    with open(csrc / "pp_kernels.cu", "a") as g:
        g.write("// a comment\n")
    ipf, dram, note, fpf = bench.load_instr_per_flight()
    assert ipf is None and "stale" in note
    monkeypatch.setenv("PP_NVCC_EXTRA", "-DPP_MIN_BLOCKS=3")  # different flags are a different kernel too
    assert bench.load_instr_per_flight()[0] is None
