// fidelity.cu -- the Turbulence-Transformer tokeniser:
//   T[m,z',y',x',c] = sum_{a,b,e<k} G[a,b,e] * Y[m, z0+k z'+a, y0+k y'+b, x0+k x'+e, c]
// a sub-domain crop C(.) followed by a normalised k^3 Gaussian filter F(.) with stride k; k = 1 is the pure crop
// (high-fidelity mode).  HBM-bound: every input voxel of the crop is read exactly once (16 bytes = the four
// variables V_x,V_y,V_z,P of one voxel), every token written once.
//
// CTA = one output row segment (fixed m, z', y'; a span of x').  Thread t owns the input column x = span_lo + t of
// all k*k input rows of that window row: k*k independent, fully coalesced 16-byte streaming loads, weighted by
// wz[a]*wy[b] in registers; then one multiply by wx[t mod k], a shared-memory exchange, and every k-th thread sums k
// neighbours and stores the token (float4 or 4 x bf16).  No input byte is touched twice and no transposes occur.
#include "kernels.cuh"

namespace ringx {
namespace {

constexpr int kThreads = 256;
constexpr int kMaxK = 32;

struct FidelityParams {
  const float4* y;
  void* tokens;
  long long stride_m, stride_z, stride_y;   // input strides in voxels (float4 units)
  int z0, y0, x0;
  int Dk, Hk, Wk;                           // output extents Dc/k, Hc/k, Wc/k
  int k;
  int span;                                 // input voxels per CTA along x (a multiple of k)
  int rows;                                 // output rows (y') per CTA: > 1 when the crop is narrower than a CTA
  float w[kMaxK];                           // normalised 1-D Gaussian weights
};

__device__ __forceinline__ float4 ldg_stream(const float4* p) {
  float4 v;
  asm volatile("ld.global.cs.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
  return v;
}

// kU = y' rows a thread works on at once (small k: keeps >= 8-16 independent 16-byte loads in flight per thread).
template <bool kOutBf16, int kU>
__global__ void __launch_bounds__(kThreads) fidelity_tokens_kernel(const __grid_constant__ FidelityParams p) {
  __shared__ float4 part[kU][kThreads];
  const int k = p.k;
  const int t = threadIdx.x;
  const int r = t / p.span;
  const int yo0 = (blockIdx.y * p.rows + r) * kU;
  const int zo = blockIdx.z % p.Dk;
  const int m = blockIdx.z / p.Dk;
  const int xin = blockIdx.x * p.span + (t - r * p.span);   // input column inside the crop
  const bool active = r < p.rows && yo0 < p.Hk && xin < p.Wk * k;
  float4 acc[kU];
#pragma unroll
  for (int u = 0; u < kU; ++u) acc[u] = make_float4(0.f, 0.f, 0.f, 0.f);
  if (active) {
    const float4* base = p.y + (long long)m * p.stride_m + (long long)(p.z0 + zo * k) * p.stride_z +
                         (long long)(p.y0 + yo0 * k) * p.stride_y + (p.x0 + xin);
    const long long ustride = (long long)k * p.stride_y;
    const int nu = min(kU, p.Hk - yo0);
    for (int a = 0; a < k; ++a) {
      const float wa = p.w[a];
      const float4* row = base + (long long)a * p.stride_z;
#pragma unroll 4
      for (int b = 0; b < k; ++b) {
        const float wab = wa * p.w[b];
        float4 v[kU];
#pragma unroll
        for (int u = 0; u < kU; ++u)
          v[u] = (u < nu) ? ldg_stream(row + (long long)b * p.stride_y + u * ustride) : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
        for (int u = 0; u < kU; ++u) {
          acc[u].x = fmaf(wab, v[u].x, acc[u].x);
          acc[u].y = fmaf(wab, v[u].y, acc[u].y);
          acc[u].z = fmaf(wab, v[u].z, acc[u].z);
          acc[u].w = fmaf(wab, v[u].w, acc[u].w);
        }
      }
    }
    const float we = p.w[t % k];
#pragma unroll
    for (int u = 0; u < kU; ++u) { acc[u].x *= we; acc[u].y *= we; acc[u].z *= we; acc[u].w *= we; }
  }
  if (k > 1) {
#pragma unroll
    for (int u = 0; u < kU; ++u) part[u][t] = acc[u];
    __syncthreads();
    if (!active || (t % k) != 0) return;
    for (int e = 1; e < k; ++e) {
#pragma unroll
      for (int u = 0; u < kU; ++u) {
        const float4 v = part[u][t + e];
        acc[u].x += v.x; acc[u].y += v.y; acc[u].z += v.z; acc[u].w += v.w;
      }
    }
  } else if (!active) {
    return;
  }
#pragma unroll
  for (int u = 0; u < kU; ++u) {
    if (yo0 + u >= p.Hk) break;
    const long long tok = (((long long)m * p.Dk + zo) * p.Hk + (yo0 + u)) * p.Wk + xin / k;
    if constexpr (kOutBf16) {
      __nv_bfloat162 lo = __floats2bfloat162_rn(acc[u].x, acc[u].y), hi = __floats2bfloat162_rn(acc[u].z, acc[u].w);
      uint2 w2;
      w2.x = *reinterpret_cast<uint32_t*>(&lo);
      w2.y = *reinterpret_cast<uint32_t*>(&hi);
      asm volatile("st.global.cs.v2.b32 [%0], {%1,%2};" ::"l"(reinterpret_cast<uint2*>(p.tokens) + tok), "r"(w2.x), "r"(w2.y) : "memory");
    } else {
      asm volatile("st.global.cs.v4.f32 [%0], {%1,%2,%3,%4};" ::"l"(reinterpret_cast<float4*>(p.tokens) + tok),
                   "f"(acc[u].x), "f"(acc[u].y), "f"(acc[u].z), "f"(acc[u].w) : "memory");
    }
  }
}

template <int kU>
void launch_u(const FidelityParams& p, dim3 grid, int out_dtype, cudaStream_t stream) {
  grid.y = (grid.y + kU - 1) / kU;
  if (out_dtype == RINGX_BF16)
    fidelity_tokens_kernel<true, kU><<<grid, kThreads, 0, stream>>>(p);
  else
    fidelity_tokens_kernel<false, kU><<<grid, kThreads, 0, stream>>>(p);
}

}  // namespace

cudaError_t launch_fidelity_tokens(const float* y, void* tokens, int M, int D, int H, int W, int z0, int y0, int x0,
                                   int Dc, int Hc, int Wc, int k, const float* w, int out_dtype, cudaStream_t stream) {
  FidelityParams p;
  p.y = reinterpret_cast<const float4*>(y);
  p.tokens = tokens;
  p.stride_y = W;
  p.stride_z = (long long)H * W;
  p.stride_m = (long long)D * H * W;
  p.z0 = z0; p.y0 = y0; p.x0 = x0;
  p.Dk = Dc / k; p.Hk = Hc / k; p.Wk = Wc / k;
  p.k = k;
  p.span = (kThreads / k) * k;
  p.rows = 1;
  if (Wc < p.span) {                        // narrow crop: several y' rows share a CTA (Wc is a multiple of k)
    p.span = Wc;
    p.rows = kThreads / Wc;
  }
  for (int i = 0; i < kMaxK; ++i) p.w[i] = i < k ? w[i] : 0.f;
  // grid.y counts y' rows here; launch_u divides it by the rows a thread handles at once
  dim3 grid((Wc + p.span - 1) / p.span, (p.Hk + p.rows - 1) / p.rows, (unsigned)(M * p.Dk));
  if (k == 1) launch_u<8>(p, grid, out_dtype, stream);
  else if (k == 2) launch_u<4>(p, grid, out_dtype, stream);
  else if (k == 3) launch_u<2>(p, grid, out_dtype, stream);
  else launch_u<1>(p, grid, out_dtype, stream);
  return cudaGetLastError();
}

}  // namespace ringx
