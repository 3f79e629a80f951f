// ddf_api.cu - C ABI entry points of libddf (include/ddf.h): model life cycle and query dispatch.
#include "ddf_common.cuh"
#include <stdlib.h>
#include <string.h>
#include <new>
#include <vector>

namespace ddf {

thread_local int g_last_cuda_error = 0;

static inline uint16_t f32_to_bf16_rne(float f) {
  uint32_t b; memcpy(&b, &f, 4);
  if ((b & 0x7F800000u) == 0x7F800000u) return (uint16_t)(b >> 16);
  return (uint16_t)((b + 0x7FFFu + ((b >> 16) & 1u)) >> 16);
}
static inline float bf16_to_f32(uint16_t h) { uint32_t b = (uint32_t)h << 16; float f; memcpy(&f, &b, 4); return f; }

static int check_layout(const ddf_layout* L) {
  if (L->struct_size != sizeof(ddf_layout) || L->version != DDF_LAYOUT_VERSION) return DDF_E_BAD_LAYOUT;
  if (L->input_kind > 1 || L->weight_dtype > 1 || L->weights_on_device > 1) return DDF_E_BAD_LAYOUT;
  if (L->n_hidden < 1 || L->n_hidden >= (uint32_t)kMaxLayers || L->width < 1) return DDF_E_BAD_LAYOUT;
  if (L->n_out < 1 || L->n_out > 2) return DDF_E_BAD_LAYOUT;
  if (L->skip_layer != -1 && (L->skip_layer < 1 || L->skip_layer >= (int32_t)L->n_hidden)) return DDF_E_BAD_LAYOUT;
  if (L->n_freq_origin > 16 || L->n_freq_dir > 16) return DDF_E_UNSUPPORTED;
  if (L->width > 16384) return DDF_E_UNSUPPORTED;
  return DDF_OK;
}

static void free_model(Model* m) {
  if (!m) return;
  tc_plan_destroy(m);
  narrow_plan_destroy(m);
  hash_plan_destroy(m);
  cudaFree(m->d_w); cudaFree(m->d_b); cudaFree(m->d_head_w);
  cudaFree(m->ws_gamma); cudaFree(m->ws_act0); cudaFree(m->ws_act1); cudaFree(m->ws_last);
  cudaFree(m->ws_dist); cudaFree(m->ws_vis);
  cudaFree(m->h2d_o); cudaFree(m->h2d_d); cudaFree(m->d2h_dist); cudaFree(m->d2h_vis);
  cudaFree(m->trace_ws); cudaFree(m->wave_ws); cudaFree(m->cam_o); cudaFree(m->cam_d);
  if (m->host_s_in) { cudaStreamDestroy(m->host_s_in); cudaStreamDestroy(m->host_s_out); for (int i = 0; i < 16; ++i) cudaEventDestroy(m->host_ev[i]); }
  (void)cudaGetLastError();
  delete m;
}

}  // namespace ddf

using namespace ddf;

extern "C" const char* ddf_status_string(int s) {
  switch (s) {
    case DDF_OK: return "ok";
    case DDF_E_INVALID_ARG: return "invalid argument";
    case DDF_E_BAD_LAYOUT: return "bad layout";
    case DDF_E_UNSUPPORTED: return "unsupported layout or device";
    case DDF_E_CUDA: return "CUDA error";
    case DDF_E_NOMEM: return "out of memory";
    case DDF_E_TOO_LARGE: return "batch exceeds the fixed capacity of this entry point";
    default: return "unknown status";
  }
}

extern "C" int ddf_last_cuda_error(void) { return g_last_cuda_error; }

// Widths the tensor-core kernels do not tile (not 64 / 128 / a multiple of 256) are served by
// padding the network with zero units up to the next such width: a padded unit has zero weights
// and zero bias, so it outputs ReLU(0) = 0 and multiplies zero weights in the next layer - every
// real accumulation sees the same terms in the same order.  Returns 0 when no padding applies.
static uint32_t padded_width(uint32_t w) {
  if (w == 64 || w == 128 || w % 256 == 0) return 0;
  if (w < 64) return 64;
  if (w < 128) return 128;
  const uint32_t up = (w + 255) / 256 * 256;
  return up <= 2048 ? up : 0;
}

static void pad_blob(const ddf_layout& L, const uint8_t* src, uint32_t w_new, std::vector<uint8_t>* dst) {
  const size_t esz = L.weight_dtype == 1 ? 2 : 4;
  const size_t E = 3 + 6 * (size_t)L.n_freq_origin + (L.input_kind == 0 ? 3 + 6 * (size_t)L.n_freq_dir : 0);
  const size_t W = L.width, Wn = w_new;
  size_t total = 0;
  for (uint32_t l = 0; l <= L.n_hidden; ++l) {
    const bool head = l == L.n_hidden;
    const size_t k0n = l == 0 ? E : Wn, k1 = ((int32_t)l == L.skip_layer) ? E : 0;
    total += (head ? L.n_out : Wn) * (k0n + k1 + 1);
  }
  dst->assign(total * esz, 0);
  size_t so = 0, dofs = 0;
  for (uint32_t l = 0; l <= L.n_hidden; ++l) {
    const bool head = l == L.n_hidden;
    const size_t k0 = l == 0 ? E : W, k0n = l == 0 ? E : Wn, k1 = ((int32_t)l == L.skip_layer) ? E : 0;
    const size_t rows = head ? L.n_out : W, rows_n = head ? L.n_out : Wn;
    for (size_t j = 0; j < rows; ++j) {
      memcpy(dst->data() + (dofs + j * (k0n + k1)) * esz, src + (so + j * (k0 + k1)) * esz, k0 * esz);
      if (k1) memcpy(dst->data() + (dofs + j * (k0n + k1) + k0n) * esz, src + (so + j * (k0 + k1) + k0) * esz, k1 * esz);
    }
    so += rows * (k0 + k1); dofs += rows_n * (k0n + k1);
    memcpy(dst->data() + dofs * esz, src + so * esz, rows * esz);           // biases
    so += rows; dofs += rows_n;
  }
}

static int create_impl(const void* weights, const ddf_layout* layout, ddf_model** out);

extern "C" int ddf_create(const void* weights, const ddf_layout* layout, ddf_model** out) {
  if (out) *out = nullptr;
  if (!weights || !layout || !out) return DDF_E_INVALID_ARG;
  int rc = check_layout(layout);
  if (rc != DDF_OK) return rc;
  uint32_t w_new = padded_width(layout->width);
  {
    // a narrow network whose weight set does not fit in shared memory (or whose encoding is wider
    // than the narrow kernel's two K blocks) goes to the wide kernel instead, padded to 256
    const uint32_t wt = w_new ? w_new : layout->width;
    if (wt == 64 || wt == 128) {
      const size_t E0 = 3 + 6 * (size_t)layout->n_freq_origin + (layout->input_kind == 0 ? 3 + 6 * (size_t)layout->n_freq_dir : 0);
      const size_t gb = (E0 + 63) / 64, hb = wt / 64;
      const size_t blocks = gb + (size_t)(layout->n_hidden - 1) * hb + (layout->skip_layer >= 1 ? gb : 0);
      const size_t smem = (gb + hb) * 16384 + blocks * wt * 128 + (size_t)(layout->n_hidden + 2) * wt * 4 + 64 + 1024;
      if (gb > 2 || smem > 232448) w_new = 256;
    }
    // padding only pays if the wide kernel will take the padded network (<= 16 layers, encoding <= 256)
    const size_t E1 = 3 + 6 * (size_t)layout->n_freq_origin + (layout->input_kind == 0 ? 3 + 6 * (size_t)layout->n_freq_dir : 0);
    if (w_new >= 256 && (layout->n_hidden > 16 || E1 > 256)) w_new = 0;
  }
  if (w_new == 0) return create_impl(weights, layout, out);
  const ddf_layout& L = *layout;
  const size_t esz = L.weight_dtype == 1 ? 2 : 4;
  const size_t E = 3 + 6 * (size_t)L.n_freq_origin + (L.input_kind == 0 ? 3 + 6 * (size_t)L.n_freq_dir : 0);
  size_t elems = 0;
  for (uint32_t l = 0; l <= L.n_hidden; ++l)
    elems += (size_t)(l == L.n_hidden ? L.n_out : L.width) * ((l == 0 ? E : L.width) + ((int32_t)l == L.skip_layer ? E : 0) + 1);
  std::vector<uint8_t> host(elems * esz), padded;
  if (L.weights_on_device) DDF_CUDA_TRY(cudaMemcpy(host.data(), weights, elems * esz, cudaMemcpyDeviceToHost));
  else memcpy(host.data(), weights, elems * esz);
  pad_blob(L, host.data(), w_new, &padded);
  ddf_layout Lp = L;
  Lp.width = w_new; Lp.weights_on_device = 0;
  return create_impl(padded.data(), &Lp, out);
}

static int create_impl(const void* weights, const ddf_layout* layout, ddf_model** out) {
  int rc;
  int dev = 0; cudaDeviceProp prop;
  DDF_CUDA_TRY(cudaGetDevice(&dev));
  DDF_CUDA_TRY(cudaGetDeviceProperties(&prop, dev));
  if (prop.major != 10) return DDF_E_UNSUPPORTED;            // sm_100a code only

  Model* m = new (std::nothrow) Model();
  if (!m) return DDF_E_NOMEM;
  memset(m, 0, sizeof(Model));
  m->lay = *layout;
  m->device = dev;
  m->sm_count = prop.multiProcessorCount;
  const ddf_layout& L = m->lay;
  m->E = 3 + 6 * (int)L.n_freq_origin + (L.input_kind == 0 ? 3 + 6 * (int)L.n_freq_dir : 0);
  m->E_pad = round_up(m->E, kKBlock);
  m->width_pad = round_up((int)L.width, kKBlock);
  m->n_layers = (int)L.n_hidden + 1;

  // walk the blob, lay out the padded device copy
  size_t blob_elems = 0, w_elems = 0, b_elems = 0;
  std::vector<size_t> src_w(m->n_layers), src_b(m->n_layers);
  std::vector<int> fan_in(m->n_layers);
  for (int l = 0; l < m->n_layers; ++l) {
    LayerDesc& d = m->layers[l];
    const bool head = (l == m->n_layers - 1);
    d.n_out = head ? (int)L.n_out : (int)L.width;
    d.k0 = (l == 0) ? m->E : (int)L.width;
    d.k0_pad = (l == 0) ? m->E_pad : m->width_pad;
    d.k1 = (l == L.skip_layer) ? m->E : 0;
    d.k1_pad = d.k1 ? m->E_pad : 0;
    d.k_pad = d.k0_pad + d.k1_pad;
    fan_in[l] = d.k0 + d.k1;
    src_w[l] = blob_elems; blob_elems += (size_t)d.n_out * fan_in[l];
    src_b[l] = blob_elems; blob_elems += (size_t)d.n_out;
    d.w_off = w_elems; w_elems += (size_t)round_up(d.n_out, 128) * d.k_pad;
    d.b_off = b_elems; b_elems += (size_t)round_up(d.n_out, 128);
  }
  m->w_elems = w_elems; m->b_elems = b_elems;

  const size_t esz = L.weight_dtype == 1 ? 2 : 4;
  std::vector<uint8_t> host_copy;
  const uint8_t* src = (const uint8_t*)weights;
  if (L.weights_on_device) {
    host_copy.resize(blob_elems * esz);
    cudaError_t e = cudaMemcpy(host_copy.data(), weights, blob_elems * esz, cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) { g_last_cuda_error = (int)e; (void)cudaGetLastError(); free_model(m); return DDF_E_CUDA; }
    src = host_copy.data();
  }
  auto src_bf16 = [&](size_t i) -> uint16_t {
    return L.weight_dtype == 1 ? ((const uint16_t*)src)[i] : f32_to_bf16_rne(((const float*)src)[i]);
  };
  auto src_f32 = [&](size_t i) -> float {
    return L.weight_dtype == 1 ? bf16_to_f32(((const uint16_t*)src)[i]) : ((const float*)src)[i];
  };
  std::vector<uint16_t> hw(w_elems, 0);
  std::vector<float> hb(b_elems, 0.0f);
  std::vector<float> hhead((size_t)L.n_out * L.width);
  for (int l = 0; l < m->n_layers; ++l) {
    const LayerDesc& d = m->layers[l];
    for (int j = 0; j < d.n_out; ++j) {
      const size_t srow = src_w[l] + (size_t)j * fan_in[l];
      uint16_t* drow = hw.data() + d.w_off + (size_t)j * d.k_pad;
      for (int k = 0; k < d.k0; ++k) drow[k] = src_bf16(srow + k);
      for (int k = 0; k < d.k1; ++k) drow[d.k0_pad + k] = src_bf16(srow + d.k0 + k);
      hb[d.b_off + j] = src_f32(src_b[l] + j);                 // biases stay fp32
      if (l == m->n_layers - 1)
        for (int k = 0; k < d.k0; ++k) hhead[(size_t)j * L.width + k] = bf16_to_f32(src_bf16(srow + k));
    }
  }
  cudaError_t e;
  if ((e = cudaMalloc(&m->d_w, w_elems * 2)) != cudaSuccess ||
      (e = cudaMalloc(&m->d_b, b_elems * 4)) != cudaSuccess ||
      (e = cudaMalloc(&m->d_head_w, hhead.size() * 4)) != cudaSuccess ||
      (e = cudaMemcpy(m->d_w, hw.data(), w_elems * 2, cudaMemcpyHostToDevice)) != cudaSuccess ||
      (e = cudaMemcpy(m->d_b, hb.data(), b_elems * 4, cudaMemcpyHostToDevice)) != cudaSuccess ||
      (e = cudaMemcpy(m->d_head_w, hhead.data(), hhead.size() * 4, cudaMemcpyHostToDevice)) != cudaSuccess) {
    g_last_cuda_error = (int)e; (void)cudaGetLastError(); free_model(m);
    return e == cudaErrorMemoryAllocation ? DDF_E_NOMEM : DDF_E_CUDA;
  }
  rc = tc_plan_create(m);
  if (rc != DDF_OK) { free_model(m); return rc; }
  if (!m->tc) {
    rc = narrow_plan_create(m, hw.data(), hb.data());
    if (rc != DDF_OK) { free_model(m); return rc; }
  }
  {
    cudaError_t es = cudaDeviceSynchronize();
    if (es != cudaSuccess) { g_last_cuda_error = (int)es; (void)cudaGetLastError(); free_model(m); return DDF_E_CUDA; }
  }
  *out = reinterpret_cast<ddf_model*>(m);
  return DDF_OK;
}

namespace ddf {
// staging of ddf_query_host (32 B per ray) and the ray workspace of ddf_query_camera / ddf_query_ao_points on models
// that read their rays from memory (24 B per ray): grown on first use, or ahead of time by ddf_reserve
static int host_reserve(Model* m, int64_t n) {
  if (n <= m->host_rows) return DDF_OK;
  cudaFree(m->h2d_o); cudaFree(m->h2d_d); cudaFree(m->d2h_dist); cudaFree(m->d2h_vis);
  m->h2d_o = m->h2d_d = m->d2h_dist = m->d2h_vis = nullptr; m->host_rows = 0;
  DDF_CUDA_TRY(cudaMalloc(&m->h2d_o, (size_t)n * 12));
  DDF_CUDA_TRY(cudaMalloc(&m->h2d_d, (size_t)n * 12));
  DDF_CUDA_TRY(cudaMalloc(&m->d2h_dist, (size_t)n * 4));
  DDF_CUDA_TRY(cudaMalloc(&m->d2h_vis, (size_t)n * 4));
  m->host_rows = n;
  if (!m->host_s_in) {
    DDF_CUDA_TRY(cudaStreamCreateWithFlags(&m->host_s_in, cudaStreamNonBlocking));
    DDF_CUDA_TRY(cudaStreamCreateWithFlags(&m->host_s_out, cudaStreamNonBlocking));
    for (int i = 0; i < 16; ++i) DDF_CUDA_TRY(cudaEventCreateWithFlags(&m->host_ev[i], cudaEventDisableTiming));
  }
  return DDF_OK;
}
static int rays_reserve(Model* m, int64_t n) {
  if (n <= m->cam_rows) return DDF_OK;
  cudaFree(m->cam_o); cudaFree(m->cam_d); m->cam_o = m->cam_d = nullptr; m->cam_rows = 0;
  DDF_CUDA_TRY(cudaMalloc(&m->cam_o, (size_t)n * 12));
  DDF_CUDA_TRY(cudaMalloc(&m->cam_d, (size_t)n * 12));
  m->cam_rows = n;
  return DDF_OK;
}
static int ao_out_reserve(Model* m, int64_t n) {
  if (n <= m->ws_out_rows) return DDF_OK;
  cudaFree(m->ws_dist); cudaFree(m->ws_vis); m->ws_dist = m->ws_vis = nullptr; m->ws_out_rows = 0;
  DDF_CUDA_TRY(cudaMalloc(&m->ws_dist, (size_t)n * 4));
  DDF_CUDA_TRY(cudaMalloc(&m->ws_vis, (size_t)n * 4));
  m->ws_out_rows = n;
  return DDF_OK;
}
}  // namespace ddf

extern "C" int ddf_reserve(ddf_model* model, uint32_t what, int64_t max_rays, int spp) {
  if (!model || max_rays < 0 || spp < 0 || (what & ~(uint32_t)DDF_RESERVE_ALL)) return DDF_E_INVALID_ARG;
  Model* m = reinterpret_cast<Model*>(model);
  { const int rc_dev = check_device(m->device); if (rc_dev != DDF_OK) return rc_dev; }
  int rc = DDF_OK;
  if (max_rays == 0) return DDF_OK;
  if ((what & DDF_RESERVE_HOST) && (rc = host_reserve(m, max_rays)) != DDF_OK) return rc;
  if ((what & DDF_RESERVE_RAYS) && (rc = rays_reserve(m, max_rays)) != DDF_OK) return rc;
  // ddf_query_ao keeps per-ray results (8 B per ray) whenever the reduce cannot be fused: no fused path, or an spp whose
  // rays do not fill whole warp fractions
  const bool ao_unfused = !has_fused_path(m) || (spp > 0 && (spp > 32 || 32 % spp != 0));
  if ((what & DDF_RESERVE_RAYS) && ao_unfused && (rc = ao_out_reserve(m, max_rays)) != DDF_OK) return rc;
  if ((what & DDF_RESERVE_TRACE) && (rc = trace_reserve(m, max_rays, 4096)) != DDF_OK) return rc;
  if ((what & DDF_RESERVE_WAVE) && (rc = wave_reserve(m, max_rays, spp)) != DDF_OK) return rc;
  // the CUDA-core path walks a batch in passes of kSimtChunkRows rays: that is all its workspace ever holds
  if (!has_fused_path(m) && (rc = ensure_workspace(m, max_rays < kSimtChunkRows ? max_rays : kSimtChunkRows)) != DDF_OK) return rc;
  return DDF_OK;
}

extern "C" int ddf_destroy(ddf_model* model) {
  if (!model) return DDF_OK;
  { const int rc_dev = check_device(reinterpret_cast<Model*>(model)->device); if (rc_dev != DDF_OK) return rc_dev; }
  cudaDeviceSynchronize();
  free_model(reinterpret_cast<Model*>(model));
  return DDF_OK;
}

extern "C" int ddf_set_path(ddf_model* model, int path) {
  if (!model || path < 0 || path > 5) return DDF_E_INVALID_ARG;
  Model* m = reinterpret_cast<Model*>(model);
  if (m->hg) return path == 0 ? DDF_OK : DDF_E_UNSUPPORTED;
  if (path == 2 && !m->tc && !m->nw) return DDF_E_UNSUPPORTED;
  if (path >= 3 && !m->tc) return DDF_E_UNSUPPORTED;
  m->path = path;
  return DDF_OK;
}

extern "C" int64_t ddf_get_info(const ddf_model* model, int which) {
  if (!model) return DDF_E_INVALID_ARG;
  const Model* m = reinterpret_cast<const Model*>(model);
  switch (which) {
    case 0: return has_fused_path(m) ? 1 : 0;
    case 1: return m->last_launches;
    case 2: return m->E;
    case 4: return m->device;
    case 3: return m->hg ? 128 : ((m->tc && m->path != 1) ? 256 : ((m->nw && m->path != 1) ? 128 : 64));
    default: return DDF_E_INVALID_ARG;
  }
}

static int run_query(Model* m, const float* o, const float* d, int64_t n, int mode_out,
                     float* out0, float* out1, void* stream) {
  if (n < 0) return DDF_E_INVALID_ARG;
  { const int rc_dev = check_device(m->device); if (rc_dev != DDF_OK) return rc_dev; }
  if (n == 0) { m->last_launches = 0; return DDF_OK; }
  if (!o || !out0 || (m->lay.input_kind == 0 && !d)) return DDF_E_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  if (has_fused_path(m)) return fused_forward(m, o, d, n, nullptr, mode_out, out0, out1, 0, 0.0f, st);
  return simt_forward(m, o, d, n, mode_out, out0, out1, st);
}

extern "C" int ddf_query(ddf_model* model, const float* origins, const float* dirs, int64_t n,
                         float* out_dist, float* out_vis, void* stream) {
  if (!model) return DDF_E_INVALID_ARG;
  return run_query(reinterpret_cast<Model*>(model), origins, dirs, n, 0, out_dist, out_vis, stream);
}

extern "C" int ddf_query_logits(ddf_model* model, const float* origins, const float* dirs, int64_t n,
                                float* out_z, void* stream) {
  if (!model) return DDF_E_INVALID_ARG;
  return run_query(reinterpret_cast<Model*>(model), origins, dirs, n, 1, out_z, nullptr, stream);
}

extern "C" int ddf_query_host(ddf_model* model, const float* origins, const float* dirs, int64_t n,
                              float* out_dist, float* out_vis, void* stream) {
  if (!model || n < 0) return DDF_E_INVALID_ARG;
  if (n == 0) return DDF_OK;
  Model* m = reinterpret_cast<Model*>(model);
  { const int rc_dev = check_device(m->device); if (rc_dev != DDF_OK) return rc_dev; }
  const bool ray = m->lay.input_kind == 0, two = m->lay.n_out == 2;
  if (!origins || !out_dist || (ray && !dirs)) return DDF_E_INVALID_ARG;
  { int rc = host_reserve(m, n); if (rc != DDF_OK) return rc; }        // a no-op after ddf_reserve(DDF_RESERVE_HOST, >= n)
  cudaStream_t st = (cudaStream_t)stream;
  // Large batches are cut into up to 8 tile-aligned chunks: the uploads run ahead on their own
  // stream, chunk i is answered on `stream` as soon as it has landed, and its results go back
  // on a third stream while chunk i+1 is being answered (results do not depend on the batching).
  int chunks = 1;
  if (n >= (1 << 18)) chunks = n >= (1 << 21) ? 8 : 4;
  if (chunks == 1) {
    DDF_CUDA_TRY(cudaMemcpyAsync(m->h2d_o, origins, (size_t)n * 12, cudaMemcpyHostToDevice, st));
    if (ray) DDF_CUDA_TRY(cudaMemcpyAsync(m->h2d_d, dirs, (size_t)n * 12, cudaMemcpyHostToDevice, st));
    int rc = run_query(m, m->h2d_o, ray ? m->h2d_d : nullptr, n, 0, m->d2h_dist, two ? m->d2h_vis : nullptr, stream);
    if (rc != DDF_OK) return rc;
    DDF_CUDA_TRY(cudaMemcpyAsync(out_dist, m->d2h_dist, (size_t)n * 4, cudaMemcpyDeviceToHost, st));
    if (two && out_vis) DDF_CUDA_TRY(cudaMemcpyAsync(out_vis, m->d2h_vis, (size_t)n * 4, cudaMemcpyDeviceToHost, st));
    DDF_CUDA_TRY(cudaStreamSynchronize(st));
    return DDF_OK;
  }
  const int64_t per = ((n + chunks - 1) / chunks + 255) / 256 * 256;
  int launches = 0;
  // the chunk pipeline; whatever it returns, no copy from or into the caller's host buffers may still be in flight
  auto pipeline = [&]() -> int {
    for (int c = 0; c < chunks; ++c) {
      const int64_t b = (int64_t)c * per, e = b + per < n ? b + per : n;
      if (b >= e) { chunks = c; break; }
      DDF_CUDA_TRY(cudaMemcpyAsync(m->h2d_o + 3 * b, origins + 3 * b, (size_t)(e - b) * 12, cudaMemcpyHostToDevice, m->host_s_in));
      if (ray) DDF_CUDA_TRY(cudaMemcpyAsync(m->h2d_d + 3 * b, dirs + 3 * b, (size_t)(e - b) * 12, cudaMemcpyHostToDevice, m->host_s_in));
      DDF_CUDA_TRY(cudaEventRecord(m->host_ev[c], m->host_s_in));
    }
    for (int c = 0; c < chunks; ++c) {
      const int64_t b = (int64_t)c * per, e = b + per < n ? b + per : n;
      DDF_CUDA_TRY(cudaStreamWaitEvent(st, m->host_ev[c], 0));
      int rc = run_query(m, m->h2d_o + 3 * b, ray ? m->h2d_d + 3 * b : nullptr, e - b, 0, m->d2h_dist + b, two ? m->d2h_vis + b : nullptr, stream);
      if (rc != DDF_OK) return rc;
      launches += m->last_launches;
      DDF_CUDA_TRY(cudaEventRecord(m->host_ev[8 + c], st));
      DDF_CUDA_TRY(cudaStreamWaitEvent(m->host_s_out, m->host_ev[8 + c], 0));
      DDF_CUDA_TRY(cudaMemcpyAsync(out_dist + b, m->d2h_dist + b, (size_t)(e - b) * 4, cudaMemcpyDeviceToHost, m->host_s_out));
      if (two && out_vis) DDF_CUDA_TRY(cudaMemcpyAsync(out_vis + b, m->d2h_vis + b, (size_t)(e - b) * 4, cudaMemcpyDeviceToHost, m->host_s_out));
    }
    return DDF_OK;
  };
  const int rc = pipeline();
  m->last_launches = launches;
  const cudaError_t e0 = cudaStreamSynchronize(m->host_s_in), e1 = cudaStreamSynchronize(st), e2 = cudaStreamSynchronize(m->host_s_out);
  if (rc != DDF_OK) { (void)cudaGetLastError(); return rc; }
  DDF_CUDA_TRY(e0); DDF_CUDA_TRY(e1); DDF_CUDA_TRY(e2);
  return DDF_OK;
}

extern "C" int ddf_query_camera(ddf_model* model, const ddf_camera* cam, int width, int height,
                                float* out_dist, float* out_vis, void* stream) {
  if (!model || !cam || width < 0 || height < 0) return DDF_E_INVALID_ARG;
  Model* m = reinterpret_cast<Model*>(model);
  { const int rc_dev = check_device(m->device); if (rc_dev != DDF_OK) return rc_dev; }
  if (m->lay.input_kind != 0) return DDF_E_INVALID_ARG;
  const int64_t n = (int64_t)width * height;
  if (n == 0) { m->last_launches = 0; return DDF_OK; }
  if (!out_dist) return DDF_E_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  if (m->hg) return hash_forward_camera(m, cam, width, height, out_dist, out_vis, st);
  int rc = rays_reserve(m, n);                                // a no-op after ddf_reserve(DDF_RESERVE_RAYS, >= n)
  if (rc != DDF_OK) return rc;
  rc = ddf_gen_camera(cam, width, height, m->cam_o, m->cam_d, stream);
  if (rc != DDF_OK) return rc;
  rc = run_query(m, m->cam_o, m->cam_d, n, 0, out_dist, out_vis, stream);
  if (rc == DDF_OK) m->last_launches += 1;
  return rc;
}

extern "C" int ddf_query_ao_points(ddf_model* model, const float* p, const float* nrm, int64_t n_pts, int spp,
                                   uint64_t seed, uint64_t rng_stream, float eps, float ao_radius, float* ao,
                                   void* stream) {
  if (!model || n_pts < 0 || spp <= 0 || n_pts * spp > 0x7fffffff) return DDF_E_INVALID_ARG;
  Model* m = reinterpret_cast<Model*>(model);
  { const int rc_dev = check_device(m->device); if (rc_dev != DDF_OK) return rc_dev; }
  if (m->lay.n_out != 2 || m->lay.input_kind != 0) return DDF_E_INVALID_ARG;
  if (n_pts == 0) { m->last_launches = 0; return DDF_OK; }
  if (!p || !nrm || !ao) return DDF_E_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  if (m->hg && spp <= 32 && 32 % spp == 0)                    // the rays never exist in memory
    return hash_forward_ao_points(m, p, nrm, n_pts, nullptr, spp, gen_key(seed, rng_stream), eps, ao_radius, ao, st);
  const int64_t n = n_pts * spp;
  int rc = rays_reserve(m, n);
  if (rc != DDF_OK) return rc;
  rc = ddf_gen_ao(p, nrm, n_pts, spp, seed, rng_stream, eps, m->cam_o, m->cam_d, stream);
  if (rc != DDF_OK) return rc;
  rc = ddf_query_ao(model, m->cam_o, m->cam_d, n_pts, spp, ao_radius, ao, stream);
  if (rc == DDF_OK) m->last_launches += 1;
  return rc;
}

extern "C" int ddf_query_ao(ddf_model* model, const float* o, const float* d, int64_t n_pts, int spp,
                            float ao_radius, float* ao, void* stream) {
  if (!model || n_pts < 0 || spp <= 0 || n_pts > (int64_t)0x7fffffff / spp) return DDF_E_INVALID_ARG;
  if (n_pts == 0) return DDF_OK;
  Model* m = reinterpret_cast<Model*>(model);
  { const int rc_dev = check_device(m->device); if (rc_dev != DDF_OK) return rc_dev; }
  if (!o || !d || !ao || m->lay.n_out != 2 || m->lay.input_kind != 0) return DDF_E_INVALID_ARG;
  const int64_t n = n_pts * spp;
  cudaStream_t st = (cudaStream_t)stream;
  if (has_fused_path(m) && spp <= 32 && 32 % spp == 0)          // a pixel's rays sit in one warp of a tile
    return fused_forward(m, o, d, n, nullptr, 2, ao, nullptr, spp, ao_radius, st);
  int rc = ao_out_reserve(m, n);
  if (rc != DDF_OK) return rc;
  rc = run_query(m, o, d, n, 0, m->ws_dist, m->ws_vis, stream);
  if (rc != DDF_OK) return rc;
  int launches = m->last_launches;
  rc = ddf_ao_reduce(m->ws_vis, m->ws_dist, n_pts, spp, ao_radius, ao, stream);
  m->last_launches = launches + 1;
  return rc;
}
