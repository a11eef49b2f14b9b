// TEST INFRASTRUCTURE, NOT PRODUCT CODE.  A host-only stand-in for the handful of CUDA runtime calls that
// paper_2405_05700_b200/csrc/pp_api.cpp makes, so that the HOST side of the library -- the batching server thread,
// the source ring, the launch slots, the hit queue, pp_submit from many threads, the multi-process front end and the
// multi-device front -- can run under ThreadSanitizer on a machine without a GPU.
// "Device" memory is host memory, every stream operation completes at once on the calling thread, events are
// always ready.  No physics here: the kernels are replaced by tests/tsan/fake_kernels.cpp.
#include <cuda_runtime.h>

#include <atomic>
#include <cstdlib>
#include <cstring>

extern "C" {

cudaError_t cudaGetDeviceCount(int* n) { *n = 1; return cudaSuccess; }
cudaError_t cudaGetDevice(int* d) { *d = 0; return cudaSuccess; }
cudaError_t cudaSetDevice(int) { return cudaSuccess; }
cudaError_t cudaDeviceGetAttribute(int* v, cudaDeviceAttr, int) { *v = 4; return cudaSuccess; }  // 4 "SMs"
const char* cudaGetErrorString(cudaError_t) { return "fake cuda error"; }
cudaError_t cudaGetLastError(void) { return cudaSuccess; }

cudaError_t cudaMalloc(void** p, size_t n) { *p = std::calloc(1, n ? n : 1); return *p ? cudaSuccess : cudaErrorMemoryAllocation; }
cudaError_t cudaFree(void* p) { std::free(p); return cudaSuccess; }
cudaError_t cudaHostAlloc(void** p, size_t n, unsigned) { *p = std::calloc(1, n ? n : 1); return *p ? cudaSuccess : cudaErrorMemoryAllocation; }
cudaError_t cudaFreeHost(void* p) { std::free(p); return cudaSuccess; }
cudaError_t cudaMemcpy(void* d, const void* s, size_t n, cudaMemcpyKind) { std::memcpy(d, s, n); return cudaSuccess; }
cudaError_t cudaMemcpyAsync(void* d, const void* s, size_t n, cudaMemcpyKind, cudaStream_t) { std::memmove(d, s, n); return cudaSuccess; }
cudaError_t cudaMemsetAsync(void* d, int v, size_t n, cudaStream_t) { std::memset(d, v, n); return cudaSuccess; }

static std::atomic<uintptr_t> g_next{16};
cudaError_t cudaStreamCreateWithFlags(cudaStream_t* s, unsigned) { *s = reinterpret_cast<cudaStream_t>(g_next.fetch_add(16)); return cudaSuccess; }
cudaError_t cudaStreamDestroy(cudaStream_t) { return cudaSuccess; }
cudaError_t cudaStreamSynchronize(cudaStream_t) { return cudaSuccess; }
cudaError_t cudaStreamWaitEvent(cudaStream_t, cudaEvent_t, unsigned) { return cudaSuccess; }
cudaError_t cudaEventCreate(cudaEvent_t* e) { *e = reinterpret_cast<cudaEvent_t>(g_next.fetch_add(16)); return cudaSuccess; }
cudaError_t cudaEventDestroy(cudaEvent_t) { return cudaSuccess; }
cudaError_t cudaEventRecord(cudaEvent_t, cudaStream_t) { return cudaSuccess; }
cudaError_t cudaEventQuery(cudaEvent_t) { return cudaSuccess; }
cudaError_t cudaEventSynchronize(cudaEvent_t) { return cudaSuccess; }
// every "launch" takes 0.01 ms and starts after the previous one: monotonic time stamps for kernel_busy_ms
cudaError_t cudaEventElapsedTime(float* ms, cudaEvent_t a, cudaEvent_t b) {
  *ms = 1.0e-3f * (float)((reinterpret_cast<uintptr_t>(b) - reinterpret_cast<uintptr_t>(a)) / 16);
  return cudaSuccess;
}

}  // extern "C"
