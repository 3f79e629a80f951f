// ddf_simt.cu - the plain CUDA-core path: encode -> per-layer tiled GEMM (bf16 operands, fp32
// accumulate, bias + ReLU, bf16 store) -> head.  It serves every layout (any width) and is the
// witness the tcgen05 path is cross-checked against on the GPU; it is not the fast path.
// Operation: include/ddf.h header comment (Eq.1).
#include "ddf_common.cuh"

namespace ddf {

// ------------------------------------------------------------------------------------------
// encode: one thread per ray, gamma row of E_pad bf16 (pad zero).  input_kind 1: point only.
__global__ void encode_kernel(const float* __restrict__ o, const float* __restrict__ d, int64_t n,
                              int input_kind, int Lo, int Ld, int E, int E_pad,
                              __nv_bfloat16* __restrict__ gamma) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  __nv_bfloat16* row = gamma + i * E_pad;
  float v[3] = { o[3 * i], o[3 * i + 1], o[3 * i + 2] };
  encode_vec_bf16(v, Lo, row);
  int m = 3 + 6 * Lo;
  if (input_kind == 0) {
    float w[3] = { d[3 * i], d[3 * i + 1], d[3 * i + 2] };
    encode_vec_bf16(w, Ld, row + m);
  }
  for (int k = E; k < E_pad; ++k) row[k] = __float2bfloat16_rn(0.0f);
}

// ------------------------------------------------------------------------------------------
// C[M][N] = ReLU( A0[M][k0] W[:, 0:k0]^T + A1[M][k1] W[:, k0_pad:k0_pad+k1]^T + b )
constexpr int BM = 64, BN = 64, BK = 16;

template <bool OUT_F32>
__global__ void __launch_bounds__(256)
simt_layer_kernel(const __nv_bfloat16* __restrict__ A0, int lda0, int k0, int k0_pad,
                  const __nv_bfloat16* __restrict__ A1, int lda1, int k1,
                  const __nv_bfloat16* __restrict__ W, int ldw, const float* __restrict__ bias,
                  int64_t M, int N, void* __restrict__ Cout, int ldc) {
  __shared__ float As[BK][BM + 1];
  __shared__ float Ws[BK][BN + 1];
  const int tx = threadIdx.x % 16, ty = threadIdx.x / 16;
  const int64_t m0 = (int64_t)blockIdx.x * BM;
  const int n0 = blockIdx.y * BN;
  float acc[4][4] = {};
  for (int seg = 0; seg < 2; ++seg) {
    const __nv_bfloat16* A = seg ? A1 : A0;
    const int lda = seg ? lda1 : lda0, kk = seg ? k1 : k0, woff = seg ? k0_pad : 0;
    if (kk == 0 || A == nullptr) continue;
    for (int kb = 0; kb < kk; kb += BK) {
      for (int e = threadIdx.x; e < BM * BK; e += 256) {
        int r = e / BK, c = e % BK;
        int64_t gm = m0 + r; int gk = kb + c;
        As[c][r] = (gm < M && gk < kk) ? __bfloat162float(A[gm * lda + gk]) : 0.0f;
        int gn = n0 + r;
        Ws[c][r] = (gn < N && gk < kk) ? __bfloat162float(W[(size_t)gn * ldw + woff + gk]) : 0.0f;
      }
      __syncthreads();
      #pragma unroll
      for (int c = 0; c < BK; ++c) {
        float a[4], w[4];
        #pragma unroll
        for (int i = 0; i < 4; ++i) { a[i] = As[c][ty * 4 + i]; w[i] = Ws[c][tx * 4 + i]; }
        #pragma unroll
        for (int i = 0; i < 4; ++i)
          #pragma unroll
          for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(a[i], w[j], acc[i][j]);
      }
      __syncthreads();
    }
  }
  #pragma unroll
  for (int i = 0; i < 4; ++i) {
    int64_t gm = m0 + ty * 4 + i;
    if (gm >= M) continue;
    #pragma unroll
    for (int j = 0; j < 4; ++j) {
      int gn = n0 + tx * 4 + j;
      if (gn >= N) continue;
      float v = fmaxf(acc[i][j] + bias[gn], 0.0f);
      if (OUT_F32) ((float*)Cout)[gm * ldc + gn] = v;
      else ((__nv_bfloat16*)Cout)[gm * ldc + gn] = __float2bfloat16_rn(v);
    }
  }
}

// ------------------------------------------------------------------------------------------
// head: one warp per ray over the fp32 last activation.  mode_out 0: heads; 1: logits.
__global__ void head_kernel(const float* __restrict__ h, int ldh, int width,
                            const float* __restrict__ Wh, const float* __restrict__ bh, int n_out,
                            int64_t n, int mode_out, float* __restrict__ out0, float* __restrict__ out1) {
  int64_t ray = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) / 32;
  int lane = threadIdx.x % 32;
  if (ray >= n) return;
  float z0 = 0.0f, z1 = 0.0f;
  for (int k = lane; k < width; k += 32) {
    float x = h[ray * ldh + k];
    z0 = fmaf(x, Wh[k], z0);
    if (n_out == 2) z1 = fmaf(x, Wh[width + k], z1);
  }
  #pragma unroll
  for (int s = 16; s > 0; s >>= 1) {
    z0 += __shfl_xor_sync(0xffffffffu, z0, s);
    z1 += __shfl_xor_sync(0xffffffffu, z1, s);
  }
  if (lane == 0) {
    z0 += bh[0];
    if (n_out == 2) z1 += bh[1];
    if (mode_out == 1) {
      out0[ray * n_out] = z0;
      if (n_out == 2) out0[ray * n_out + 1] = z1;
    } else if (n_out == 2) {
      out0[ray] = softplus_f(z0);
      if (out1) out1[ray] = sigmoid_f(z1);
    } else {
      out0[ray] = z0;
    }
  }
}

// ------------------------------------------------------------------------------------------
int ensure_workspace(Model* m, int64_t rows) {
  if (rows <= m->ws_rows) return DDF_OK;
  cudaFree(m->ws_gamma); cudaFree(m->ws_act0); cudaFree(m->ws_act1); cudaFree(m->ws_last);
  m->ws_gamma = m->ws_act0 = m->ws_act1 = nullptr; m->ws_last = nullptr; m->ws_rows = 0;
  DDF_CUDA_TRY(cudaMalloc(&m->ws_gamma, (size_t)rows * m->E_pad * 2));
  DDF_CUDA_TRY(cudaMalloc(&m->ws_act0, (size_t)rows * m->width_pad * 2));
  DDF_CUDA_TRY(cudaMalloc(&m->ws_act1, (size_t)rows * m->width_pad * 2));
  DDF_CUDA_TRY(cudaMalloc(&m->ws_last, (size_t)rows * m->width_pad * 4));
  m->ws_rows = rows;
  return DDF_OK;
}

int simt_forward(Model* m, const float* o, const float* d, int64_t n, int mode_out,
                 float* out0, float* out1, cudaStream_t st) {
  const int64_t kChunk = kSimtChunkRows;
  int rc = ensure_workspace(m, n < kChunk ? n : kChunk);
  if (rc != DDF_OK) return rc;
  const ddf_layout& L = m->lay;
  int launches = 0;
  for (int64_t base = 0; base < n; base += kChunk) {
    int64_t cn = (n - base < kChunk) ? n - base : kChunk;
    encode_kernel<<<(unsigned)((cn + 127) / 128), 128, 0, st>>>(
        o + 3 * base, d ? d + 3 * base : nullptr, cn, (int)L.input_kind, (int)L.n_freq_origin,
        (int)L.n_freq_dir, m->E, m->E_pad, m->ws_gamma);
    ++launches;
    const __nv_bfloat16* in = m->ws_gamma; int ld_in = m->E_pad;
    for (int l = 0; l < (int)L.n_hidden; ++l) {
      const LayerDesc& ld = m->layers[l];
      bool last = (l == (int)L.n_hidden - 1);
      __nv_bfloat16* outb = (l % 2 == 0) ? m->ws_act0 : m->ws_act1;
      dim3 grid((unsigned)((cn + BM - 1) / BM), (unsigned)((ld.n_out + BN - 1) / BN));
      const __nv_bfloat16* A1 = ld.k1 ? m->ws_gamma : nullptr;
      if (last)
        simt_layer_kernel<true><<<grid, 256, 0, st>>>(in, ld_in, ld.k0, ld.k0_pad, A1, m->E_pad, ld.k1,
            m->d_w + ld.w_off, ld.k_pad, m->d_b + ld.b_off, cn, ld.n_out, m->ws_last, m->width_pad);
      else
        simt_layer_kernel<false><<<grid, 256, 0, st>>>(in, ld_in, ld.k0, ld.k0_pad, A1, m->E_pad, ld.k1,
            m->d_w + ld.w_off, ld.k_pad, m->d_b + ld.b_off, cn, ld.n_out, outb, m->width_pad);
      ++launches;
      in = outb; ld_in = m->width_pad;
    }
    const LayerDesc& hd = m->layers[L.n_hidden];
    float* o0 = (mode_out == 1) ? out0 + base * L.n_out : out0 + base;
    float* o1 = out1 ? out1 + base : nullptr;
    head_kernel<<<(unsigned)((cn * 32 + 255) / 256), 256, 0, st>>>(
        m->ws_last, m->width_pad, (int)L.width, m->d_head_w, m->d_b + hd.b_off, (int)L.n_out, cn,
        mode_out, o0, o1);
    ++launches;
  }
  DDF_CUDA_TRY(cudaGetLastError());
  m->last_launches = launches;
  return DDF_OK;
}

}  // namespace ddf
