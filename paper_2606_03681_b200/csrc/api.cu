// C ABI of libtabattn (include/tabattn.h): argument validation and kernel dispatch.
// No device allocation, no host synchronisation; everything is enqueued on the caller's stream.
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include "../../include/tabattn.h"
#include "kernels.h"

#include <atomic>

using tabattn::Shape;

namespace tabattn {
static std::atomic<uint64_t> g_launches{0};
void count_launch(int n) { g_launches.fetch_add((uint64_t)n, std::memory_order_relaxed); }
}  // namespace tabattn

namespace {

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

// Validate the shape and translate it for the kernels.  Returns TABATTN_OK or the error.
tabattn_status check_shape(const tabattn_shape* sh, bool item, Shape* out) {
  if (!sh) return TABATTN_ERR_INVALID_ARG;
  if (sh->B < 1 || sh->R < 1 || sh->C < 1 || sh->H < 1 || sh->dh < 1) return TABATTN_ERR_INVALID_ARG;
  if (sh->dh != 16 && sh->dh != 32 && sh->dh != 64) return TABATTN_ERR_UNSUPPORTED;
  const long long cells = (long long)sh->B * sh->R * sh->C;
  if (cells >= (1LL << 31) || (long long)sh->H * sh->dh > TABATTN_MAX_D) return TABATTN_ERR_UNSUPPORTED;
  if (item) {
    if (!sh->n_train) return TABATTN_ERR_INVALID_ARG;
    if (sh->n_train_host)
      for (int b = 0; b < sh->B; ++b)
        if (sh->n_train_host[b] < 1 || sh->n_train_host[b] > sh->R) return TABATTN_ERR_INVALID_ARG;
  }
  out->B = sh->B; out->R = sh->R; out->C = sh->C; out->H = sh->H; out->dh = sh->dh;
  out->n_train = sh->n_train;
  out->col_valid = sh->col_valid;
  out->scale = sh->softmax_scale > 0.f ? sh->softmax_scale : 1.0f / sqrtf((float)sh->dh);
  if (!item && !tabattn::feature_shape_supported(*out)) return TABATTN_ERR_UNSUPPORTED;
  return TABATTN_OK;
}

// The calling thread's current device must be sm_100 (per-device, thread-safe: device.cu).
tabattn_status check_device() {
  const tabattn::DeviceInfo* di = tabattn::current_device();
  if (!di) return TABATTN_ERR_CUDA;
  return di->cc_major == 10 ? TABATTN_OK : TABATTN_ERR_UNSUPPORTED;
}

// Outputs may not alias any other argument (tabattn.h): equal base pointers are rejected.  (Partial
// overlaps of distinct allocations cannot be told from here and stay the caller's responsibility.)
template <size_t NO, size_t NI>
bool aliased(const void* const (&outs)[NO], const void* const (&ins)[NI]) {
  for (size_t i = 0; i < NO; ++i) {
    for (size_t j = i + 1; j < NO; ++j)
      if (outs[i] == outs[j]) return true;
    for (size_t j = 0; j < NI; ++j)
      if (outs[i] == ins[j]) return true;
  }
  return false;
}

template <typename... P>
bool all_ok(P... p) {
  const void* v[] = {p...};
  for (const void* x : v)
    if (!x || !aligned16(x)) return false;
  return true;
}

tabattn_status from_cuda(cudaError_t e) { return e == cudaSuccess ? TABATTN_OK : TABATTN_ERR_CUDA; }

tabattn_status check_ws(size_t need, const void* ws, size_t ws_bytes) {
  if (need == 0) return TABATTN_OK;
  if (!ws || ws_bytes < need || !aligned16(ws)) return TABATTN_ERR_WORKSPACE;
  return TABATTN_OK;
}

}  // namespace

extern "C" {

int tabattn_version(void) { return TABATTN_VERSION; }

uint64_t tabattn_launch_count(void) { return tabattn::g_launches.load(std::memory_order_relaxed); }

const char* tabattn_status_string(tabattn_status st) {
  switch (st) {
    case TABATTN_OK: return "ok";
    case TABATTN_ERR_INVALID_ARG: return "invalid argument";
    case TABATTN_ERR_UNSUPPORTED: return "unsupported shape or device";
    case TABATTN_ERR_WORKSPACE: return "workspace missing, misaligned or too small";
    case TABATTN_ERR_CUDA: return "CUDA error";
  }
  return "unknown status";
}

size_t tabattn_workspace_bytes(const tabattn_shape* sh, int op) {
  Shape s;
  if (!sh || op < 0 || op > 3) return 0;
  tabattn_shape tmp = *sh;
  static const int32_t dummy = 1;
  if (!tmp.n_train) tmp.n_train = &dummy;  // sizes do not depend on the values
  tmp.n_train_host = nullptr;
  if (check_shape(&tmp, op >= 2, &s) != TABATTN_OK) return 0;
  switch (op) {
    case TABATTN_OP_ITEM_BWD: return tabattn::item_bwd_workspace_bytes(s);
    case TABATTN_OP_FEATURE_FWD:
    case TABATTN_OP_FEATURE_BWD: return tabattn::feature_workspace_bytes(s);
    default: return 0;
  }
}

tabattn_status tabattn_feature_fwd(const tabattn_shape* sh, const void* Q, const void* K, const void* V, void* O,
                                   float* LSE, void* ws, size_t ws_bytes, tabattn_stream stream) {
  Shape s;
  tabattn_status st = check_shape(sh, false, &s);
  if (st != TABATTN_OK) return st;
  if (!all_ok(Q, K, V, (const void*)O, (const void*)LSE)) return TABATTN_ERR_INVALID_ARG;
  {
    const void* const outs[] = {O, LSE};
    const void* const ins[] = {Q, K, V};
    if (aliased(outs, ins)) return TABATTN_ERR_INVALID_ARG;
  }
  // the workspace is only touched when a column mask is given (per-table geometry, a0)
  if (s.col_valid && (st = check_ws(tabattn::feature_workspace_bytes(s), ws, ws_bytes)) != TABATTN_OK) return st;
  if ((st = check_device()) != TABATTN_OK) return st;
  return from_cuda(tabattn::launch_feature_fwd(s, Q, K, V, O, LSE, ws, (cudaStream_t)stream));
}

tabattn_status tabattn_feature_bwd(const tabattn_shape* sh, const void* Q, const void* K, const void* V,
                                   const void* O, const void* dO, const float* LSE, void* dQ, void* dK, void* dV,
                                   void* ws, size_t ws_bytes, tabattn_stream stream) {
  Shape s;
  tabattn_status st = check_shape(sh, false, &s);
  if (st != TABATTN_OK) return st;
  if (!all_ok(Q, K, V, O, dO, (const void*)LSE, (const void*)dQ, (const void*)dK, (const void*)dV))
    return TABATTN_ERR_INVALID_ARG;
  {
    const void* const outs[] = {dQ, dK, dV};
    const void* const ins[] = {Q, K, V, O, dO, LSE};
    if (aliased(outs, ins)) return TABATTN_ERR_INVALID_ARG;
  }
  if (s.col_valid && (st = check_ws(tabattn::feature_workspace_bytes(s), ws, ws_bytes)) != TABATTN_OK) return st;
  if ((st = check_device()) != TABATTN_OK) return st;
  return from_cuda(tabattn::launch_feature_bwd(s, Q, K, V, O, dO, LSE, dQ, dK, dV, ws, (cudaStream_t)stream));
}

tabattn_status tabattn_item_fwd(const tabattn_shape* sh, const void* Q, const void* K, const void* V, void* O,
                                float* LSE, void* ws, size_t ws_bytes, tabattn_stream stream) {
  Shape s;
  tabattn_status st = check_shape(sh, true, &s);
  if (st != TABATTN_OK) return st;
  (void)ws; (void)ws_bytes;
  if (!all_ok(Q, K, V, (const void*)O, (const void*)LSE)) return TABATTN_ERR_INVALID_ARG;
  {
    const void* const outs[] = {O, LSE};
    const void* const ins[] = {Q, K, V};
    if (aliased(outs, ins)) return TABATTN_ERR_INVALID_ARG;
  }
  if ((st = check_device()) != TABATTN_OK) return st;
  return from_cuda(tabattn::launch_item_fwd(s, Q, K, V, O, LSE, 0, s.R, (cudaStream_t)stream));
}

tabattn_status tabattn_feature_fwd_infer(const tabattn_shape* sh, const void* Q, const void* K, const void* V, void* O,
                                         int32_t row0, int32_t row1, void* ws, size_t ws_bytes,
                                         tabattn_stream stream) {
  Shape s;
  tabattn_status st = check_shape(sh, false, &s);
  if (st != TABATTN_OK) return st;
  if (!all_ok(Q, K, V, (const void*)O) || row0 < 0 || row1 <= row0 || row1 > s.R) return TABATTN_ERR_INVALID_ARG;
  {
    const void* const outs[] = {O};
    const void* const ins[] = {Q, K, V};
    if (aliased(outs, ins)) return TABATTN_ERR_INVALID_ARG;
  }
  if (s.col_valid && (st = check_ws(tabattn::feature_workspace_bytes(s), ws, ws_bytes)) != TABATTN_OK) return st;
  if ((st = check_device()) != TABATTN_OK) return st;
  return from_cuda(tabattn::launch_feature_fwd_infer(s, Q, K, V, O, row0, row1, ws, (cudaStream_t)stream));
}

tabattn_status tabattn_item_fwd_infer(const tabattn_shape* sh, const void* Q, const void* K, const void* V, void* O,
                                      int32_t row0, int32_t row1, void* ws, size_t ws_bytes, tabattn_stream stream) {
  Shape s;
  tabattn_status st = check_shape(sh, true, &s);
  if (st != TABATTN_OK) return st;
  (void)ws; (void)ws_bytes;
  if (!all_ok(Q, K, V, (const void*)O) || row0 < 0 || row1 <= row0 || row1 > s.R) return TABATTN_ERR_INVALID_ARG;
  {
    const void* const outs[] = {O};
    const void* const ins[] = {Q, K, V};
    if (aliased(outs, ins)) return TABATTN_ERR_INVALID_ARG;
  }
  if ((st = check_device()) != TABATTN_OK) return st;
  return from_cuda(tabattn::launch_item_fwd(s, Q, K, V, O, nullptr, row0, row1, (cudaStream_t)stream));
}

tabattn_status tabattn_item_bwd(const tabattn_shape* sh, const void* Q, const void* K, const void* V,
                                const void* O, const void* dO, const float* LSE, void* dQ, void* dK, void* dV,
                                void* ws, size_t ws_bytes, tabattn_stream stream) {
  Shape s;
  tabattn_status st = check_shape(sh, true, &s);
  if (st != TABATTN_OK) return st;
  if (!all_ok(Q, K, V, O, dO, (const void*)LSE, (const void*)dQ, (const void*)dK, (const void*)dV))
    return TABATTN_ERR_INVALID_ARG;
  {
    const void* const outs[] = {dQ, dK, dV, ws};
    const void* const ins[] = {Q, K, V, O, dO, LSE};
    if (aliased(outs, ins)) return TABATTN_ERR_INVALID_ARG;
  }
  if ((st = check_ws(tabattn::item_bwd_workspace_bytes(s), ws, ws_bytes)) != TABATTN_OK) return st;
  if ((st = check_device()) != TABATTN_OK) return st;
  return from_cuda(tabattn::launch_item_bwd(s, Q, K, V, O, dO, LSE, dQ, dK, dV, static_cast<float*>(ws),
                                            (cudaStream_t)stream));
}

}  // extern "C"
