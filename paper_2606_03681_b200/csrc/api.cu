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
    // masked item calls pack (b, c) into 16 + 16 bits (the a0 column list)
    if (sh->col_valid && (sh->B > 65535 || sh->C > 65535)) return TABATTN_ERR_UNSUPPORTED;
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
    case TABATTN_OP_ITEM_FWD: return tabattn::item_fwd_workspace_bytes(s);
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
  if (!all_ok(Q, K, V, (const void*)O, (const void*)LSE)) return TABATTN_ERR_INVALID_ARG;
  {
    const void* const outs[] = {O, LSE};
    const void* const ins[] = {Q, K, V};
    if (aliased(outs, ins)) return TABATTN_ERR_INVALID_ARG;
  }
  // the workspace is only touched when a column mask is given (the a0 column list)
  if (s.col_valid && (st = check_ws(tabattn::item_fwd_workspace_bytes(s), ws, ws_bytes)) != TABATTN_OK) return st;
  if ((st = check_device()) != TABATTN_OK) return st;
  return from_cuda(tabattn::launch_item_fwd(s, Q, K, V, O, LSE, 0, s.R, ws, (cudaStream_t)stream));
}

tabattn_status tabattn_item_fwd_noalloc(const tabattn_shape* sh, const void* Q, const void* K, const void* V, void* O,
                                        float* LSE, tabattn_stream stream) {
  Shape s;
  tabattn_status st = check_shape(sh, true, &s);
  if (st != TABATTN_OK) return st;
  if (!all_ok(Q, K, V, (const void*)O, (const void*)LSE)) return TABATTN_ERR_INVALID_ARG;
  {
    const void* const outs[] = {O, LSE};
    const void* const ins[] = {Q, K, V};
    if (aliased(outs, ins)) return TABATTN_ERR_INVALID_ARG;
  }
  // the column list of a masked call must fit the library's own device array (TABATTN_NOALLOC_MAX_BC pairs)
  if (s.col_valid && ((long long)s.B * s.C > TABATTN_NOALLOC_MAX_BC ||
                      tabattn::item_fwd_workspace_bytes(s) > tabattn::item_fwd_noalloc_capacity()))
    return TABATTN_ERR_WORKSPACE;
  if ((st = check_device()) != TABATTN_OK) return st;
  return from_cuda(tabattn::launch_item_fwd_noalloc(s, Q, K, V, O, LSE, (cudaStream_t)stream));
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
  if (!all_ok(Q, K, V, (const void*)O) || row0 < 0 || row1 <= row0 || row1 > s.R) return TABATTN_ERR_INVALID_ARG;
  {
    const void* const outs[] = {O};
    const void* const ins[] = {Q, K, V};
    if (aliased(outs, ins)) return TABATTN_ERR_INVALID_ARG;
  }
  if (s.col_valid && (st = check_ws(tabattn::item_fwd_workspace_bytes(s), ws, ws_bytes)) != TABATTN_OK) return st;
  if ((st = check_device()) != TABATTN_OK) return st;
  return from_cuda(tabattn::launch_item_fwd(s, Q, K, V, O, nullptr, row0, row1, ws, (cudaStream_t)stream));
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

// ---- sub-blocks -------------------------------------------------------------------

namespace {
bool block_dims_ok(int e, int hidden) { return e >= 64 && e <= 1024 && e % 64 == 0 && (hidden == 0 || (hidden >= 64 && hidden % 64 == 0)); }
float or_default(float v, float d) { return v > 0.f ? v : d; }
}  // namespace

size_t tabattn_attn_block_workspace_bytes(const tabattn_shape* sh, int32_t axis, int32_t backward) {
  Shape s;
  if (!sh || (axis != 0 && axis != 1)) return 0;
  tabattn_shape tmp = *sh;
  static const int32_t dummy = 1;
  if (!tmp.n_train) tmp.n_train = &dummy;
  tmp.n_train_host = nullptr;
  if (check_shape(&tmp, axis == 1, &s) != TABATTN_OK) return 0;
  const tabattn::DeviceInfo* di = tabattn::current_device();
  const int sms = di ? di->num_sms : 148;
  return backward ? tabattn::attn_block_bwd_ws_bytes(s, axis, sms)
                  : (axis == 0 ? tabattn::feature_workspace_bytes(s) : tabattn::item_fwd_workspace_bytes(s));
}

tabattn_status tabattn_attn_block_fwd(const tabattn_shape* sh, int32_t axis, float alpha, float eps, const void* x,
                                      const void* g, const void* Wqkv, const void* Wo, void* y,
                                      const tabattn_attn_saved* sv, void* ws, size_t ws_bytes, tabattn_stream stream) {
  Shape s;
  if (axis != 0 && axis != 1) return TABATTN_ERR_INVALID_ARG;
  tabattn_status st = check_shape(sh, axis == 1, &s);
  if (st != TABATTN_OK) return st;
  if (!block_dims_ok(s.H * s.dh, 0)) return TABATTN_ERR_UNSUPPORTED;
  if (!sv || !all_ok(x, g, Wqkv, Wo, (const void*)y, (const void*)sv->h, (const void*)sv->rstd, (const void*)sv->q,
                     (const void*)sv->k, (const void*)sv->v, (const void*)sv->o, (const void*)sv->lse))
    return TABATTN_ERR_INVALID_ARG;
  {
    const void* const outs[] = {y, sv->h, sv->rstd, sv->q, sv->k, sv->v, sv->o, sv->lse};
    const void* const ins[] = {x, g, Wqkv, Wo};
    if (aliased(outs, ins)) return TABATTN_ERR_INVALID_ARG;
  }
  if (s.col_valid && (st = check_ws(axis == 0 ? tabattn::feature_workspace_bytes(s) : tabattn::item_fwd_workspace_bytes(s), ws,
                                    ws_bytes)) != TABATTN_OK)
    return st;
  if ((st = check_device()) != TABATTN_OK) return st;
  return from_cuda(tabattn::launch_attn_block_fwd(s, axis, or_default(alpha, 1.f), or_default(eps, 1e-6f), x, g, Wqkv,
                                                  Wo, y, sv->h, sv->rstd, sv->q, sv->k, sv->v, sv->o, sv->lse, ws,
                                                  (cudaStream_t)stream));
}

tabattn_status tabattn_attn_block_bwd(const tabattn_shape* sh, int32_t axis, float alpha, const void* x, const void* g,
                                      const void* Wqkv, const void* Wo, const tabattn_attn_saved* sv, const void* dy,
                                      void* dx, float* dg, float* dWqkv, float* dWo, void* ws, size_t ws_bytes,
                                      tabattn_stream stream) {
  Shape s;
  if (axis != 0 && axis != 1) return TABATTN_ERR_INVALID_ARG;
  tabattn_status st = check_shape(sh, axis == 1, &s);
  if (st != TABATTN_OK) return st;
  if (!block_dims_ok(s.H * s.dh, 0)) return TABATTN_ERR_UNSUPPORTED;
  if (!sv || !all_ok(x, g, Wqkv, Wo, dy, (const void*)dx, (const void*)dg, (const void*)dWqkv, (const void*)dWo,
                     (const void*)sv->h, (const void*)sv->rstd, (const void*)sv->q, (const void*)sv->k,
                     (const void*)sv->v, (const void*)sv->o, (const void*)sv->lse))
    return TABATTN_ERR_INVALID_ARG;
  {
    const void* const outs[] = {dx, dg, dWqkv, dWo, ws};
    const void* const ins[] = {x, g, Wqkv, Wo, dy, sv->h, sv->rstd, sv->q, sv->k, sv->v, sv->o, sv->lse};
    if (aliased(outs, ins)) return TABATTN_ERR_INVALID_ARG;
  }
  if ((st = check_device()) != TABATTN_OK) return st;
  const tabattn::DeviceInfo* di = tabattn::current_device();
  if ((st = check_ws(tabattn::attn_block_bwd_ws_bytes(s, axis, di->num_sms), ws, ws_bytes)) != TABATTN_OK) return st;
  return from_cuda(tabattn::launch_attn_block_bwd(s, axis, or_default(alpha, 1.f), x, g, Wqkv, Wo, sv->h, sv->rstd,
                                                  sv->q, sv->k, sv->v, sv->o, sv->lse, dy, dx, dg, dWqkv, dWo, ws,
                                                  ws_bytes, (cudaStream_t)stream));
}

size_t tabattn_mlp_workspace_bytes(int64_t cells, int32_t e, int32_t hidden) {
  if (cells < 1 || cells >= (1LL << 31) || !block_dims_ok(e, hidden) || hidden == 0) return 0;
  const tabattn::DeviceInfo* di = tabattn::current_device();
  return tabattn::block_ws_bytes(cells, e, hidden, di ? di->num_sms : 148);
}

tabattn_status tabattn_mlp_fwd(int64_t cells, int32_t e, int32_t hidden, float alpha, float eps, const void* x,
                               const void* g, const void* W1, const void* W2, void* y, const tabattn_mlp_saved* sv,
                               tabattn_stream stream) {
  if (cells < 1) return TABATTN_ERR_INVALID_ARG;
  if (cells >= (1LL << 31) || !block_dims_ok(e, hidden) || hidden == 0) return TABATTN_ERR_UNSUPPORTED;
  if (!sv || !all_ok(x, g, W1, W2, (const void*)y, (const void*)sv->h, (const void*)sv->rstd, (const void*)sv->u,
                     (const void*)sv->a))
    return TABATTN_ERR_INVALID_ARG;
  {
    const void* const outs[] = {y, sv->h, sv->rstd, sv->u, sv->a};
    const void* const ins[] = {x, g, W1, W2};
    if (aliased(outs, ins)) return TABATTN_ERR_INVALID_ARG;
  }
  tabattn_status st = check_device();
  if (st != TABATTN_OK) return st;
  return from_cuda(tabattn::launch_mlp_fwd(cells, e, hidden, or_default(alpha, 1.f), or_default(eps, 1e-6f), x, g, W1,
                                           W2, y, sv->h, sv->rstd, sv->u, sv->a, (cudaStream_t)stream));
}

tabattn_status tabattn_mlp_bwd(int64_t cells, int32_t e, int32_t hidden, float alpha, const void* x, const void* g,
                               const void* W1, const void* W2, const tabattn_mlp_saved* sv, const void* dy, void* dx,
                               float* dg, float* dW1, float* dW2, void* ws, size_t ws_bytes, tabattn_stream stream) {
  if (cells < 1) return TABATTN_ERR_INVALID_ARG;
  if (cells >= (1LL << 31) || !block_dims_ok(e, hidden) || hidden == 0) return TABATTN_ERR_UNSUPPORTED;
  if (!sv || !all_ok(x, g, W1, W2, dy, (const void*)dx, (const void*)dg, (const void*)dW1, (const void*)dW2,
                     (const void*)sv->h, (const void*)sv->rstd, (const void*)sv->u, (const void*)sv->a))
    return TABATTN_ERR_INVALID_ARG;
  {
    const void* const outs[] = {dx, dg, dW1, dW2, ws};
    const void* const ins[] = {x, g, W1, W2, dy, sv->h, sv->rstd, sv->u, sv->a};
    if (aliased(outs, ins)) return TABATTN_ERR_INVALID_ARG;
  }
  tabattn_status st = check_device();
  if (st != TABATTN_OK) return st;
  if ((st = check_ws(tabattn_mlp_workspace_bytes(cells, e, hidden), ws, ws_bytes)) != TABATTN_OK) return st;
  return from_cuda(tabattn::launch_mlp_bwd(cells, e, hidden, or_default(alpha, 1.f), x, g, W1, W2, sv->h, sv->rstd,
                                           sv->u, sv->a, dy, dx, dg, dW1, dW2, ws, ws_bytes, (cudaStream_t)stream));
}

size_t tabattn_newton_schulz_workspace_bytes(int32_t nb, int32_t m, int32_t n) {
  if (nb < 1 || m < 8 || n < m || (m & 7) || (n & 7)) return 0;
  return tabattn::newton_schulz_ws_bytes(nb, m, n);
}

tabattn_status tabattn_newton_schulz(int32_t nb, int32_t m, int32_t n, const void* G, void* X, int32_t steps, void* ws,
                                     size_t ws_bytes, tabattn_stream stream) {
  if (nb < 1 || m < 1 || n < 1 || steps < 0) return TABATTN_ERR_INVALID_ARG;
  if (m < 8 || n < m || (m & 7) || (n & 7) || steps > 64) return TABATTN_ERR_UNSUPPORTED;
  if (!all_ok(G, (const void*)X) || G == X) return TABATTN_ERR_INVALID_ARG;
  tabattn_status st = check_ws(tabattn::newton_schulz_ws_bytes(nb, m, n), ws, ws_bytes);
  if (st != TABATTN_OK) return st;
  if ((st = check_device()) != TABATTN_OK) return st;
  // Muon's quintic coefficients (Jordan et al. 2024b, as in modded-nanogpt)
  return from_cuda(tabattn::launch_newton_schulz(nb, m, n, G, X, steps, 3.4445f, -4.7750f, 2.0315f, 1e-7f, ws,
                                                 (cudaStream_t)stream));
}

}  // extern "C"
