// Host-side per-device state of libtabattn: everything the launch paths cache is keyed by the CUDA
// device ordinal and safe to use from several host threads (include/tabattn.h: "re-entrant across
// host threads on different streams with different workspaces").  Not exported.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

#include <atomic>
#include <stdint.h>

namespace tabattn {

constexpr int kMaxDevices = 64;

struct DeviceInfo {
  int ordinal;    // cudaGetDevice() of the calling thread
  int cc_major;   // compute capability major (10 = sm_100)
  int num_sms;
};

// Properties of the calling thread's current device, queried once per ordinal (std::call_once).
// Returns nullptr if the runtime cannot name a device or the ordinal is >= kMaxDevices.
const DeviceInfo* current_device();

// cudaFuncSetAttribute(MaxDynamicSharedMemorySize) is per device: one of these per kernel
// instantiation, one bit per device ordinal.  A lost race repeats an idempotent call.
struct SmemAttr {
  std::atomic<uint64_t> done{0};
  template <typename Kern>
  cudaError_t ensure(Kern kern, int bytes, int dev) {
    const uint64_t bit = 1ull << (dev & 63);
    if (done.load(std::memory_order_acquire) & bit) return cudaSuccess;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e == cudaSuccess) done.fetch_or(bit, std::memory_order_release);
    return e;
  }
};

// CUtensorMap over a [cells][H][dh]-shaped bf16 tensor, cached per (device, base pointer, geometry):
// encoding one costs ~1 us of driver time and every item call needs 3-8 of them.
//   kind 0: item view, dims (dh, H, C, R, B), box (dh, 1, 1, box_rows, 1)   -- one (b, c, h) sequence
//   kind 1: feature view, dims (dh, H, C, B*R), box (dh, 1, box_c, box_rows) -- rows x columns of one head
// Swizzle span = one row of dh bf16 (32/64/128 B).  Out-of-range coordinates are zero-filled on load
// and clipped on store.  Returns false if the driver entry point is missing or the encode fails.
bool get_tensor_map(CUtensorMap* out, int kind, const void* base, int B, int R, int C, int H, int dh, int box_rows,
                    int box_c);

}  // namespace tabattn
