// Internal interface between the host side of the library (pp_api.cpp) and its kernels
// (pp_kernels.cu).  Not part of the public ABI.
#pragma once
#include <atomic>
#include <cstddef>
#include <cstdint>
#include <cuda_runtime.h>

#include "../../include/pp.h"
#include "pp_types.h"

namespace pp {

uint64_t kernel_launch_count();

cudaError_t launch_ingest(const pp_source* d_s, const uint32_t* d_ev, const uint32_t* d_sid, uint32_t sid_base, uint32_t n,
                          float yield, SrcRec* d_out, unsigned int* d_overflow, cudaStream_t st);
cudaError_t launch_scan(const SrcRec* d_src, uint32_t n, unsigned long long* d_cum, cudaStream_t st);
// tiles + cum_rel for photons [g_begin, ...) of a scanned batch; also clears *d_status for the launch that follows
cudaError_t launch_tiles(const unsigned long long* d_cum, uint32_t n_src, unsigned long long g_begin, uint32_t n_tiles,
                         uint32_t tile_photons, uint32_t* d_tile_src, uint32_t* d_cum_rel, Status* d_status,
                         cudaStream_t st);
// scan + tiles + cum_rel + status in one single-CTA kernel: small launches only (n_src, n_tiles <= kPrologueMax)
constexpr uint32_t kPrologueMax = 4096;
cudaError_t launch_prologue(const SrcRec* d_src, uint32_t n_src, unsigned long long* d_cum, unsigned long long g_begin,
                            uint32_t n_tiles, uint32_t tile_photons, uint32_t* d_tile_src, uint32_t* d_cum_rel,
                            Status* d_status, cudaStream_t st);
cudaError_t launch_propagate(const LaunchParams& P, bool brute, bool fates, int grid, size_t smem, cudaStream_t st);
cudaError_t propagate_occupancy(bool brute, bool fates, size_t smem, int* blocks_per_sm);
int propagate_warps_per_block();  // warps of one CTA of the propagation kernel

// What pp_run_resident_noalloc (pp_kernels.cu) needs to know about a handle (defined in pp_api.cpp, where pp_handle
// is): a copy of the launch template with the medium, the geometry and the optional physics filled in, and how the
// handle launches the propagation kernel.  Returns PP_OK, or the handle's sticky error / PP_E_STATE after shutdown.
struct HandleLaunchInfo {
  LaunchParams base;
  int device, grid;
  size_t smem;
  bool brute;
  float photons_per_GeV;
};
int handle_launch_info(pp_handle* h, HandleLaunchInfo* out);
int handle_fail(pp_handle* h, int code, const char* msg);  // records msg for pp_last_error; returns code

// Step 1 on the host (same arithmetic as the device's, exact in fp64).
inline unsigned long long host_photon_count(float energy, float yield) {
  // floor(E y + 1/2) by truncation: the same integer for a non-negative argument, and no call into libm on a host
  // compiler's baseline x86-64 (this runs once per submitted source: 4e7 times a second behind the IPC front end)
  const double n = (double)energy * (double)yield + 0.5;
  if (!(n >= 1.0)) return 0ull;
  if (n >= 1.8e19) return ~0ull;
  return (unsigned long long)n;
}

}  // namespace pp
