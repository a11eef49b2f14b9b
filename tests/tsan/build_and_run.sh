#!/bin/bash
# ThreadSanitizer pass over the HOST side of the library: pp_api.cpp, pp_ipc.cpp and pp_multi.cpp
# built with -fsanitize=thread against a fake CUDA runtime and fake kernels (this directory), driven by driver.cpp.
# Usage: tests/tsan/build_and_run.sh [out_dir]   (exit code 0 = no data race, all checks passed)
set -e
HERE=$(cd "$(dirname "$0")" && pwd)
ROOT=$(cd "$HERE/../.." && pwd)
OUT=${1:-$(mktemp -d)}
CUDA_INC=${CUDA_HOME:-/usr/local/cuda}/include
g++ -std=c++17 -O1 -g -fsanitize=thread -fno-omit-frame-pointer -pthread -I"$CUDA_INC" \
    "$ROOT"/paper_2405_05700_b200/csrc/pp_api.cpp "$ROOT"/paper_2405_05700_b200/csrc/pp_ipc.cpp \
    "$ROOT"/paper_2405_05700_b200/csrc/pp_multi.cpp "$HERE"/fake_cuda.cpp "$HERE"/fake_kernels.cpp "$HERE"/driver.cpp \
    -o "$OUT"/pp_tsan_driver -lrt
TSAN_OPTIONS="exitcode=66 halt_on_error=1 second_deadlock_stack=1" "$OUT"/pp_tsan_driver
