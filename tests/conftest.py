import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")
    config.addinivalue_line("markers", "slow: longer statistical test")
    # a hung kernel or a dead-locked server must fail the run, not stall it: with pytest-timeout installed every test
    # gets 15 minutes unless the command line says otherwise ('thread' method: works while blocked in a C call)
    if config.pluginmanager.hasplugin("timeout") and not getattr(config.option, "timeout", None):
        config.option.timeout = 900.0
        config.option.timeout_method = "thread"
        config._env_timeout, config._env_timeout_method = 900.0, "thread"  # (the plugin has read its settings already)
    # build the CUDA library (nvcc cross-compiles without a GPU) and the oracle; both builders compare modification
    # times, so an up-to-date binary is left alone and a stale one is never what the tests exercise
    from paper_2405_05700_b200 import build as pp_build
    pp_build.build()
    from oracle import oracle as O
    O.build()
    build_echo_backend()
    build_guard_library()


GUARD_LIB = os.path.join(ROOT, "tests", "libpp_guard.so")


def build_guard_library() -> str:
    """tests/libpp_guard.so: the library compiled with -DPP_GUARD (guard zones behind every piece of the device
    workspace, checked by the host after every launch; index checks inside the kernel: csrc/pp_guard.cuh).  Test
    infrastructure standing in for compute-sanitizer; tests/test_gpu_guard.py runs against it in a process of its own."""
    from paper_2405_05700_b200 import build as pp_build
    return pp_build.build(out=GUARD_LIB, defines=("PP_GUARD",))


ECHO_LIB = os.path.join(ROOT, "tests", "libpp_echo.so")


def build_echo_backend() -> str:
    """tests/libpp_echo.so: the host-only back end the CPU tests of the multi-process front end plug into
    pp_ipc_server_create_backend (test infrastructure; not part of libpp.so)."""
    import subprocess
    src = os.path.join(ROOT, "tests", "echo_backend.cpp")
    deps = [src, os.path.join(ROOT, "include", "pp_ipc.h"), os.path.join(ROOT, "include", "pp.h")]
    if not os.path.exists(ECHO_LIB) or any(os.path.getmtime(d) > os.path.getmtime(ECHO_LIB) for d in deps):
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-o", ECHO_LIB, src])
    return ECHO_LIB


def pytest_collection_modifyitems(config, items):
    """GPU tests fail loudly (not skip) on a GPU box without the extension; on a CPU box they are
    deselected by ``-m "not gpu"``.  If someone runs the whole suite on a CPU box, skip them."""
    try:
        import torch
        has_gpu = torch.cuda.is_available()
    except Exception:  # pragma: no cover
        has_gpu = False
    if has_gpu:
        return
    skip = pytest.mark.skip(reason="no CUDA device")
    for item in items:
        if "gpu" in item.keywords:
            item.add_marker(skip)
