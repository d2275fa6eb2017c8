// attn_f32.cu -- fp32 chunk attention on plain FFMA (no tensor cores): config C1 of BASELINE.json.
// tcgen05 kind::tf32 keeps 10 mantissa bits and would give ~2.5e-5 error on O at N=1024, over the
// 1e-5 bar, so the fp32 path is SIMT.  One chunk pass computes, for every query
// row, loc_out = softmax(scale q.K_c^T) V_c and loc_lse with an online softmax over
// groups of 8 keys.  It is 0.27 GFLOP at C1: correctness path, not a performance path.
#include "kernels.cuh"

namespace ringx {
namespace {

constexpr int kThreads = 128;
constexpr int kKeysPerTile = 32;
constexpr int kGroup = 8;

// kSplit threads share one query row; each owns 64 of the d dims of q and of the output.
template <int kSplit>
__global__ void __launch_bounds__(kThreads)
attn_chunk_f32_kernel(const float* __restrict__ q, const float* __restrict__ k, const float* __restrict__ v,
                      float* __restrict__ o_out, float* __restrict__ lse_out, int Nq, int nk_stride, int k_off, int nk,
                      float scale) {
  constexpr int d = 64 * kSplit;
  constexpr int kRows = kThreads / kSplit;
  __shared__ __align__(16) float sK[kKeysPerTile][d];
  __shared__ __align__(16) float sV[kKeysPerTile][d];

  const int bh = blockIdx.y;
  const int row = blockIdx.x * kRows + threadIdx.x / kSplit;
  const int part = threadIdx.x % kSplit;
  const float* qrow = q + ((size_t)bh * Nq + row) * d + part * 64;
  const float* kbase = k + ((size_t)bh * nk_stride + k_off) * d;
  const float* vbase = v + ((size_t)bh * nk_stride + k_off) * d;

  float qr[64], acc[64];
#pragma unroll
  for (int c = 0; c < 64; ++c) {
    qr[c] = qrow[c];
    acc[c] = 0.f;
  }
  float m = -CUDART_INF_F, l = 0.f;

  for (int k0 = 0; k0 < nk; k0 += kKeysPerTile) {
    __syncthreads();
    for (int i = threadIdx.x; i < kKeysPerTile * d / 4; i += kThreads) {
      reinterpret_cast<float4*>(&sK[0][0])[i] = reinterpret_cast<const float4*>(kbase + (size_t)k0 * d)[i];
      reinterpret_cast<float4*>(&sV[0][0])[i] = reinterpret_cast<const float4*>(vbase + (size_t)k0 * d)[i];
    }
    __syncthreads();
    for (int g = 0; g < kKeysPerTile; g += kGroup) {
      float s[kGroup];
#pragma unroll
      for (int j = 0; j < kGroup; ++j) {
        float dot = 0.f;
#pragma unroll
        for (int c = 0; c < 64; ++c) dot = fmaf(qr[c], sK[g + j][part * 64 + c], dot);
        if (kSplit == 2) dot += __shfl_xor_sync(0xffffffffu, dot, 1);
        s[j] = dot * scale;
      }
      float gm = s[0];
#pragma unroll
      for (int j = 1; j < kGroup; ++j) gm = fmaxf(gm, s[j]);
      const float m_new = fmaxf(m, gm);
      const float corr = expf(m - m_new);           // exp(-inf) = 0 on the first group
      l *= corr;
#pragma unroll
      for (int c = 0; c < 64; ++c) acc[c] *= corr;
#pragma unroll
      for (int j = 0; j < kGroup; ++j) {
        const float p = expf(s[j] - m_new);
        l += p;
#pragma unroll
        for (int c = 0; c < 64; ++c) acc[c] = fmaf(p, sV[g + j][part * 64 + c], acc[c]);
      }
      m = m_new;
    }
  }
  const float inv = 1.0f / l;
  float* orow = o_out + ((size_t)bh * Nq + row) * d + part * 64;
#pragma unroll
  for (int c = 0; c < 64; c += 4)
    *reinterpret_cast<float4*>(orow + c) = make_float4(acc[c] * inv, acc[c + 1] * inv, acc[c + 2] * inv, acc[c + 3] * inv);
  if (part == 0) lse_out[(size_t)bh * Nq + row] = m + logf(l);
}

}  // namespace

cudaError_t launch_attn_chunk_f32(const float* q, const float* k, const float* v, float* o_out, float* lse_out, int BH,
                                  int Nq, int nk_stride, int k_off, int nk, int d, float scale, cudaStream_t stream) {
  if (d == 64) {
    dim3 grid(Nq / kThreads, BH);
    attn_chunk_f32_kernel<1><<<grid, kThreads, 0, stream>>>(q, k, v, o_out, lse_out, Nq, nk_stride, k_off, nk, scale);
  } else {
    dim3 grid(Nq / (kThreads / 2), BH);
    attn_chunk_f32_kernel<2><<<grid, kThreads, 0, stream>>>(q, k, v, o_out, lse_out, Nq, nk_stride, k_off, nk, scale);
  }
  count_launch();
  return cudaGetLastError();
}

}  // namespace ringx
