// ddf_trace.cu - sphere tracing of an SDF MLP, the comparison point of PAPER.md:19 / 112 and
// Table IV: "a sequential loop, and each iteration is a full evaluation".
// Step rule and the traced function s(p) = (|p| - R) + alpha MLP(p): include/ddf.h.
// Per step: points kernel -> MLP forward (same kernels as ddf_query) -> update kernel.  With
// early_exit the live rays are compacted into an index list whose length stays on the device; the
// compaction is stable (per-block survivor counts -> the one-block scan of ddf_wave.cu -> scatter),
// so the list, and with it which rays share an MMA tile, is the same run to run.
// omega > 1: over-relaxed steps with the safe fall-back of reading A19' (include/ddf.h).
#include "ddf_common.cuh"
#include <math.h>

namespace ddf {

struct TraceWs {
  float* pts;        // [n][3] compacted points of the current step
  float* z;          // [n]    MLP output for them
  int32_t* idx[2];   // live-ray lists (ping-pong)
  int64_t* counts;   // [max_steps + 2] live count entering each step; last = total evals
  uint8_t* done;     // [n]
  float* relax;      // [3][n] over-relaxation state per ray: factor still in use, previous t, previous s (NaN: none)
  int32_t* block_counts;   // survivors per 256-entry block of the live list, then their exclusive scan
};

__global__ void trace_init_kernel(int64_t n, float* t, uint8_t* hit, int32_t* steps, uint8_t* done,
                                  int32_t* idx0, int64_t* counts, int n_counts,
                                  float* trace_p, float* trace_s, int max_steps, float* relax, float omega, int64_t relax_stride) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i == 0) { for (int k = 0; k < n_counts; ++k) counts[k] = 0; counts[0] = n; }
  const float qnan = __int_as_float(0x7fc00000);
  if (i < n) { t[i] = 0.0f; hit[i] = 0; steps[i] = 0; done[i] = 0; idx0[i] = (int32_t)i; }
  if (i < n && omega > 1.0f) { relax[i] = omega; relax[relax_stride + i] = 0.0f; relax[2 * relax_stride + i] = qnan; }
  if (trace_s) for (int64_t k = i; k < n * max_steps; k += (int64_t)gridDim.x * blockDim.x) trace_s[k] = qnan;
  if (trace_p) for (int64_t k = i; k < n * max_steps * 3; k += (int64_t)gridDim.x * blockDim.x) trace_p[k] = qnan;
}

__global__ void trace_points_kernel(const int32_t* __restrict__ idx, const int64_t* __restrict__ count,
                                    const float* __restrict__ o, const float* __restrict__ d,
                                    const float* __restrict__ t, float* __restrict__ pts, int64_t* total) {
  int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t cnt = *count;
  if (j == 0 && total) *total += cnt;
  if (j >= cnt) return;
  int64_t i = idx[j];
  float tt = t[i];
  #pragma unroll
  for (int a = 0; a < 3; ++a) pts[3 * j + a] = fmaf(tt, d[3 * i + a], o[3 * i + a]);
}

// One step of the rule for every entry of the live list.  With early_exit it also counts, per 256-entry block, the rays
// that stay alive (block_counts); trace_compact_kernel then writes them to the next list in the same order.
__global__ void __launch_bounds__(256)
trace_update_kernel(const int32_t* __restrict__ idx_in, const int64_t* __restrict__ count_in,
                    const float* __restrict__ pts, const float* __restrict__ z,
                    int step, sdf_trace_params prm,
                    float* __restrict__ t, uint8_t* __restrict__ hit, int32_t* __restrict__ steps,
                    uint8_t* __restrict__ done, int32_t* __restrict__ block_counts,
                    float* __restrict__ trace_p, float* __restrict__ trace_s,
                    float* __restrict__ relax, int64_t relax_stride) {
  int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  bool alive = false;
  if (j < *count_in) {
    int64_t i = idx_in[j];
    if (!done[i]) {                                      // fixed-step mode keeps finished rays in the list
      float px = pts[3 * j], py = pts[3 * j + 1], pz = pts[3 * j + 2];
      float n2 = fmaf(pz, pz, fmaf(py, py, px * px));
      float s = fmaf(prm.alpha, z[j], sqrtf(n2) - prm.base_radius);
      steps[i] = step + 1;
      if (trace_s) trace_s[i * prm.max_steps + step] = s;
      if (trace_p) { float* q = trace_p + (i * prm.max_steps + step) * 3; q[0] = px; q[1] = py; q[2] = pz; }
      bool fin = false;
      const float tcur = t[i];
      float om = 1.0f;
      bool redo = false;
      if (prm.omega > 1.0f) {
        om = relax[i];
        const float tp = relax[relax_stride + i], sp = relax[2 * relax_stride + i];     // sp is NaN when there is no previous point
        if (om > 1.0f && __fadd_rn(fabsf(s), fabsf(sp)) < __fsub_rn(tcur, tp)) {
          // the spheres at the previous and at this point do not touch: the relaxed step may have jumped a surface.
          // Back to where the plain step would have gone, and no relaxation for this ray from here on.
          const float tt = __fadd_rn(tp, sp);
          t[i] = tt; relax[i] = 1.0f; relax[2 * relax_stride + i] = __int_as_float(0x7fc00000);
          if (tt > prm.t_max || tt < 0.0f) fin = true;
          redo = true;
        }
      }
      if (!redo) {
        if (fabsf(s) < prm.eps) { hit[i] = 1; fin = true; }
        else {
          if (prm.omega > 1.0f) { relax[relax_stride + i] = tcur; relax[2 * relax_stride + i] = s; }
          float tt = fmaf(om, s, tcur);                  // om == 1: exactly tcur + s
          t[i] = tt;
          if (tt > prm.t_max || tt < 0.0f) fin = true;
        }
      }
      if (fin) done[i] = 1;
      alive = !fin;
    }
  }
  if (prm.early_exit) {
    const int c = __syncthreads_count(alive);
    if (threadIdx.x == 0) block_counts[blockIdx.x] = c;
  }
}

// entries of the live list whose ray is not done, in list order, to idx_out at block_offsets[block] + rank in block
__global__ void __launch_bounds__(256)
trace_compact_kernel(const int32_t* __restrict__ idx_in, const int64_t* __restrict__ count_in,
                     const uint8_t* __restrict__ done, const int32_t* __restrict__ block_offsets,
                     int32_t* __restrict__ idx_out) {
  __shared__ int32_t warp_base[8];
  const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  int32_t i = 0;
  bool alive = false;
  if (j < *count_in) { i = idx_in[j]; alive = !done[i]; }
  const uint32_t m = __ballot_sync(0xffffffffu, alive);
  if (lane == 0) warp_base[warp] = __popc(m);
  __syncthreads();
  if (threadIdx.x == 0) {
    int32_t run = 0;
    for (int w = 0; w < 8; ++w) { const int32_t c = warp_base[w]; warp_base[w] = run; run += c; }
  }
  __syncthreads();
  if (alive) idx_out[(int64_t)block_offsets[blockIdx.x] + warp_base[warp] + __popc(m & ((1u << lane) - 1u))] = i;
}

}  // namespace ddf

using namespace ddf;

namespace ddf {
// workspace of sdf_sphere_trace for n rays and S steps: pts 12n, z 4n, idx 2*4n, relaxation state 12n, done n,
// counts, survivor counts per 256-entry block
static size_t trace_need(int64_t n, int S, size_t* rows) {
  const size_t a = (size_t)((n + 63) / 64 * 64);
  if (rows) *rows = a;
  return a * 12 + a * 4 + a * 8 + a * 12 + a + (size_t)(S + 2) * 8 + ((a + 255) / 256) * 4 + 256;
}
int trace_reserve(Model* m, int64_t n, int S) {
  const size_t need = trace_need(n, S, nullptr);
  if (need <= m->trace_ws_bytes) return DDF_OK;
  cudaFree(m->trace_ws); m->trace_ws = nullptr; m->trace_ws_bytes = 0;
  DDF_CUDA_TRY(cudaMalloc(&m->trace_ws, need));
  m->trace_ws_bytes = need;
  return DDF_OK;
}
}  // namespace ddf

extern "C" int sdf_sphere_trace(ddf_model* model, const float* o, const float* d, int64_t n,
                                const sdf_trace_params* prm, float* out_t, uint8_t* out_hit,
                                int32_t* out_steps, float* trace_p, float* trace_s, int64_t* total_evals,
                                void* stream) {
  if (!model || !prm || n < 0 || n > 0x7fffffff) return DDF_E_INVALID_ARG;
  Model* m = reinterpret_cast<Model*>(model);
  { const int rc_dev = check_device(m->device); if (rc_dev != DDF_OK) return rc_dev; }
  if (m->lay.input_kind != 1 || m->lay.n_out != 1) return DDF_E_INVALID_ARG;
  if (prm->max_steps < 1 || prm->max_steps > 4096) return DDF_E_INVALID_ARG;
  if (!(prm->omega >= 0.0f && prm->omega < 2.0f)) return DDF_E_INVALID_ARG;     // also refuses NaN
  if (n == 0) return DDF_OK;
  if (!o || !d || !out_t || !out_hit || !out_steps) return DDF_E_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  const int S = prm->max_steps;
  size_t a;
  (void)trace_need(n, S, &a);
  { int rc = trace_reserve(m, n, S); if (rc != DDF_OK) return rc; }    // a no-op after ddf_reserve(DDF_RESERVE_TRACE)
  uint8_t* base = (uint8_t*)m->trace_ws;
  TraceWs w;
  w.pts = (float*)base;                 base += a * 12;
  w.z = (float*)base;                   base += a * 4;
  w.idx[0] = (int32_t*)base;            base += a * 4;
  w.idx[1] = (int32_t*)base;            base += a * 4;
  w.relax = (float*)base;               base += a * 12;
  w.counts = (int64_t*)base;            base += (size_t)(S + 2) * 8;
  w.block_counts = (int32_t*)base;      base += ((a + 255) / 256) * 4;
  w.done = base;

  const unsigned nb = (unsigned)((n + 255) / 256);
  trace_init_kernel<<<nb, 256, 0, st>>>(n, out_t, out_hit, out_steps, w.done, w.idx[0], w.counts, S + 2,
                                        trace_p, trace_s, S, w.relax, prm->omega, (int64_t)a);
  int launches = 1;
  const bool use_tc = has_fused_path(m);
  int64_t live = n;
  for (int step = 0; step < S; ++step) {
    const int cur = prm->early_exit ? (step & 1) : 0;
    int64_t* cnt_in = prm->early_exit ? w.counts + step : w.counts;          // fixed mode: always n
    int64_t* cnt_out = w.counts + step + 1;
    const unsigned gb = (unsigned)((live + 255) / 256);
    trace_points_kernel<<<gb, 256, 0, st>>>(w.idx[cur], cnt_in, o, d, out_t, w.pts, w.counts + S + 1);
    int rc;
    if (use_tc) rc = fused_forward(m, w.pts, nullptr, live, cnt_in, 1, w.z, nullptr, 0, 0.0f, st);
    else rc = simt_forward(m, w.pts, nullptr, live, 1, w.z, nullptr, st);
    if (rc != DDF_OK) return rc;
    launches += 1 + m->last_launches;
    trace_update_kernel<<<gb, 256, 0, st>>>(w.idx[cur], cnt_in, w.pts, w.z, step, *prm, out_t, out_hit,
                                           out_steps, w.done, w.block_counts, trace_p, trace_s, w.relax, (int64_t)a);
    ++launches;
    if (prm->early_exit) {
      if ((rc = scan_block_counts(w.block_counts, (int64_t)gb, cnt_out, st)) != DDF_OK) return rc;
      trace_compact_kernel<<<gb, 256, 0, st>>>(w.idx[cur], cnt_in, w.done, w.block_counts, w.idx[cur ^ 1]);
      launches += 2;
    }
    if (prm->early_exit && !use_tc) {
      // the SIMT path sizes its grids on the host: read the live count back (synchronises)
      DDF_CUDA_TRY(cudaMemcpyAsync(&live, cnt_out, 8, cudaMemcpyDeviceToHost, st));
      DDF_CUDA_TRY(cudaStreamSynchronize(st));
      if (live == 0) break;
    }
  }
  if (total_evals)
    DDF_CUDA_TRY(cudaMemcpyAsync(total_evals, w.counts + S + 1, 8, cudaMemcpyDeviceToDevice, st));
  DDF_CUDA_TRY(cudaGetLastError());
  m->last_launches = launches;
  return DDF_OK;
}
