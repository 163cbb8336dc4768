// Per-device host state (device.h): device properties, CUtensorMap cache.
// The driver entry point is fetched through the runtime (no link-time dependency on libcuda).
#include "device.h"

#include <cudaTypedefs.h>
#include <string.h>

#include <mutex>

namespace tabattn {

namespace {

struct DevSlot {
  std::once_flag once;
  DeviceInfo info;
  bool ok = false;
};
DevSlot g_dev[kMaxDevices];

PFN_cuTensorMapEncodeTiled_v12000 encode_fn() {
  static PFN_cuTensorMapEncodeTiled_v12000 fn = []() -> PFN_cuTensorMapEncodeTiled_v12000 {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess)
      return nullptr;
    return reinterpret_cast<PFN_cuTensorMapEncodeTiled_v12000>(p);
  }();   // (function-local static: initialised once, thread-safe)
  return fn;
}

struct MapKey {
  const void* base;
  int32_t dev, kind, B, R, C, H, dh, box_rows, box_c;
  bool operator==(const MapKey& o) const { return memcmp(this, &o, sizeof(MapKey)) == 0; }
};
struct MapEntry {
  MapKey key;
  CUtensorMap map;
  bool used = false;
};
constexpr int kMapSlots = 512;   // direct-mapped, 4 ways
std::mutex g_map_mu;
MapEntry g_maps[kMapSlots];
uint32_t g_map_clock = 0;

uint32_t hash_key(const MapKey& k) {
  uint64_t h = reinterpret_cast<uintptr_t>(k.base) * 0x9E3779B97F4A7C15ull;
  const int32_t v[9] = {k.dev, k.kind, k.B, k.R, k.C, k.H, k.dh, k.box_rows, k.box_c};
  for (int32_t x : v) h = (h ^ (uint32_t)x) * 0x100000001B3ull;
  return (uint32_t)(h >> 32);
}

bool encode(CUtensorMap* map, const MapKey& k) {
  auto fn = encode_fn();
  if (!fn) return false;
  const cuuint64_t d = (cuuint64_t)k.H * k.dh;
  const CUtensorMapSwizzle sw = k.dh == 64   ? CU_TENSOR_MAP_SWIZZLE_128B
                                : k.dh == 32 ? CU_TENSOR_MAP_SWIZZLE_64B
                                             : CU_TENSOR_MAP_SWIZZLE_32B;
  cuuint32_t estr[5] = {1, 1, 1, 1, 1};
  CUresult r;
  if (k.kind == 0) {
    cuuint64_t dims[5] = {(cuuint64_t)k.dh, (cuuint64_t)k.H, (cuuint64_t)k.C, (cuuint64_t)k.R, (cuuint64_t)k.B};
    cuuint64_t strides[4] = {(cuuint64_t)k.dh * 2, d * 2, (cuuint64_t)k.C * d * 2, (cuuint64_t)k.R * k.C * d * 2};
    cuuint32_t box[5] = {(cuuint32_t)k.dh, 1, 1, (cuuint32_t)k.box_rows, 1};
    r = fn(map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 5, const_cast<void*>(k.base), dims, strides, box, estr,
           CU_TENSOR_MAP_INTERLEAVE_NONE, sw, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  } else {
    cuuint64_t dims[4] = {(cuuint64_t)k.dh, (cuuint64_t)k.H, (cuuint64_t)k.C, (cuuint64_t)k.B * k.R};
    cuuint64_t strides[3] = {(cuuint64_t)k.dh * 2, d * 2, (cuuint64_t)k.C * d * 2};
    cuuint32_t box[4] = {(cuuint32_t)k.dh, 1, (cuuint32_t)k.box_c, (cuuint32_t)k.box_rows};
    r = fn(map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, const_cast<void*>(k.base), dims, strides, box, estr,
           CU_TENSOR_MAP_INTERLEAVE_NONE, sw, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  }
  return r == CUDA_SUCCESS;
}

}  // namespace

const DeviceInfo* current_device() {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return nullptr;
  DevSlot& s = g_dev[dev];
  std::call_once(s.once, [&]() {
    s.info.ordinal = dev;
    s.ok = cudaDeviceGetAttribute(&s.info.cc_major, cudaDevAttrComputeCapabilityMajor, dev) == cudaSuccess &&
           cudaDeviceGetAttribute(&s.info.num_sms, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess &&
           s.info.num_sms > 0;
  });
  return s.ok ? &s.info : nullptr;
}

bool get_tensor_map(CUtensorMap* out, int kind, const void* base, int B, int R, int C, int H, int dh, int box_rows,
                    int box_c) {
  const DeviceInfo* di = current_device();
  if (!di) return false;
  MapKey k;
  memset(&k, 0, sizeof(k));   // (padding bytes take part in the comparison)
  k.base = base; k.dev = di->ordinal; k.kind = kind; k.B = B; k.R = R; k.C = C; k.H = H; k.dh = dh;
  k.box_rows = box_rows; k.box_c = box_c;
  const uint32_t set = (hash_key(k) % (kMapSlots / 4)) * 4;
  {
    std::lock_guard<std::mutex> lock(g_map_mu);
    for (int w = 0; w < 4; ++w)
      if (g_maps[set + w].used && g_maps[set + w].key == k) {
        *out = g_maps[set + w].map;
        return true;
      }
  }
  CUtensorMap m;
  if (!encode(&m, k)) return false;
  {
    std::lock_guard<std::mutex> lock(g_map_mu);
    int victim = -1;
    for (int w = 0; w < 4 && victim < 0; ++w)
      if (!g_maps[set + w].used) victim = w;
    if (victim < 0) victim = (int)(g_map_clock++ & 3);
    g_maps[set + victim].key = k;
    g_maps[set + victim].map = m;
    g_maps[set + victim].used = true;
  }
  *out = m;
  return true;
}

}  // namespace tabattn
