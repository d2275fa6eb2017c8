// attn_f32_split_sm100.cu -- the fp32 path of the chunk attention ON THE TENSOR CORES: config C1
// of BASELINE.json (fp32, <= 1e-5 on O) cannot run on kind::tf32 (10 mantissa bits: ~2.5e-5 on O at N = 1024), and the
// bf16 MMA keeps 8.  But an fp32 number is EXACTLY the sum of three bf16 numbers,
//     x = hi + mid + lo,   hi = bf16(x),  mid = bf16(x - hi),  lo = bf16(x - hi - mid)      (both differences are exact),
// so a product of two fp32 operands is the sum of nine bf16 x bf16 products, each of which the tensor core forms exactly
// and accumulates in fp32.  Keeping the six terms of order <= 2^-16 (hi hi, hi mid, mid hi, hi lo, lo hi, mid mid) leaves
// a relative error of ~3 * 2^-24 per product -- fp32 accuracy from bf16 MMAs:
//     S   = Q K_c^T      = sum over the six (Q_a, K_b) pairs of  Q_a K_b^T               (Eq. 4)
//     O_c = P V_c        = sum over the six (P_a, V_b) pairs of  P_a V_b                 (Eq. 1)
// with P = exp(scale S - m) computed in fp32 registers and split the same way.  The small terms are issued first, so that
// they are added before the large ones.  Measured on C1: max |O - O_ref| 5.6e-7 (a plain FFMA kernel: ~1e-6; kind::tf32: ~2.5e-5).
//
// This is a correctness path (0.27 GFLOP at C1), so the kernel is the simplest correct one: a CTA = 128 query rows, 128
// threads (thread = query row = TMEM lane), no warp specialisation, no pipeline: per 128-key tile
//   all threads: K_j fp32 -> three 128B-swizzled bf16 tiles in shared memory;  thread 0: the S MMAs;  all: wait;
//   all threads: V_j -> the same shared memory;  online softmax on S from TMEM, P -> three bf16 tiles in TMEM;
//   thread 0: the P V MMAs;  all: wait.
// TMEM columns: S [0,128) fp32, P_hi / P_mid / P_lo [128,192) [192,256) [256,320) bf16, O [320, 320 + d) fp32.
#include "kernels.cuh"

namespace ringx {
namespace {

using namespace ptx;

constexpr int kTile = 128;
constexpr int kPanelBytes = 128 * 128;            // [128 rows][64 bf16], 128B-swizzled
constexpr uint32_t tS = 0, tP = 128, tO = 320;    // TMEM columns; P split a at tP + 64 a

template <int kD>
struct SplitCfg {
  static constexpr int kPanels = kD / 64;
  static constexpr int kTileBytes = kPanels * kPanelBytes;          // one bf16 [128, d] tile
  static constexpr int kSmemBytes = 1024 + 6 * kTileBytes + 64;     // Q_hi Q_mid Q_lo | KV_hi KV_mid KV_lo | barrier, slot
};

// x -> (hi, mid, lo) as three bf16 bit patterns
__device__ __forceinline__ void split3(float x, uint16_t& hi, uint16_t& mid, uint16_t& lo) {
  const __nv_bfloat16 h = __float2bfloat16_rn(x);
  const float r1 = x - __bfloat162float(h);
  const __nv_bfloat16 m = __float2bfloat16_rn(r1);
  const float r2 = r1 - __bfloat162float(m);
  const __nv_bfloat16 l = __float2bfloat16_rn(r2);
  hi = __bfloat16_as_ushort(h);
  mid = __bfloat16_as_ushort(m);
  lo = __bfloat16_as_ushort(l);
}

// One fp32 row [d] of a [128, d] tile -> row `r` of the three swizzled bf16 tiles at base + a * tile_bytes.
// Element (r, c) of a panel sits at r * 128 + ((c / 8) ^ (r & 7)) * 16 + (c % 8) * 2  (the TMA / UMMA 128-byte swizzle).
template <int kD>
__device__ __forceinline__ void split_row_to_smem(const float* __restrict__ src, uint8_t* base, int r) {
  using Cfg = SplitCfg<kD>;
#pragma unroll
  for (int c8 = 0; c8 < kD / 8; ++c8) {                   // 8 columns = one 16-byte chunk of the bf16 row
    const float4 x0 = __ldg(reinterpret_cast<const float4*>(src + c8 * 8));
    const float4 x1 = __ldg(reinterpret_cast<const float4*>(src + c8 * 8 + 4));
    const float x[8] = {x0.x, x0.y, x0.z, x0.w, x1.x, x1.y, x1.z, x1.w};
    uint16_t h[8], m[8], l[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) split3(x[i], h[i], m[i], l[i]);
    const int panel = c8 >> 3, chunk = c8 & 7;
    uint8_t* dst = base + panel * kPanelBytes + r * 128 + ((chunk ^ (r & 7)) << 4);
    auto pack = [](const uint16_t (&u)[8], int i) { return static_cast<uint32_t>(u[i]) | (static_cast<uint32_t>(u[i + 1]) << 16); };
    st_shared_v4(dst, pack(h, 0), pack(h, 2), pack(h, 4), pack(h, 6));
    st_shared_v4(dst + Cfg::kTileBytes, pack(m, 0), pack(m, 2), pack(m, 4), pack(m, 6));
    st_shared_v4(dst + 2 * Cfg::kTileBytes, pack(l, 0), pack(l, 2), pack(l, 4), pack(l, 6));
  }
}

// the six operand pairs (a, b) with a + b <= 2 (0 = hi, 1 = mid, 2 = lo), smallest products first:
//   (mid, mid) (hi, lo) (lo, hi) (hi, mid) (mid, hi) (hi, hi)
__device__ __forceinline__ constexpr int pair_a(int t) { return t == 0 ? 1 : t == 1 ? 0 : t == 2 ? 2 : t == 3 ? 0 : t == 4 ? 1 : 0; }
__device__ __forceinline__ constexpr int pair_b(int t) { return t == 0 ? 1 : t == 1 ? 2 : t == 2 ? 0 : t == 3 ? 1 : 0; }

template <int kD>
__global__ void __launch_bounds__(kTile, 1)
attn_chunk_f32_split_kernel(const float* __restrict__ q, const float* __restrict__ k, const float* __restrict__ v,
                            float* __restrict__ o_out, float* __restrict__ lse_out, int Nq, int nk_stride, int k_off,
                            int nk, float scale) {
  using Cfg = SplitCfg<kD>;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t* sQ = smem;                                   // [3][tile]
  uint8_t* sKV = smem + 3 * Cfg::kTileBytes;            // [3][tile]: K_j, then V_j
  uint64_t* bar = reinterpret_cast<uint64_t*>(sKV + 3 * Cfg::kTileBytes);
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bar + 1);

  const int warp = threadIdx.x >> 5;
  const int r = threadIdx.x;                            // my query row of the tile = TMEM lane; also the K/V row I convert
  const int bh = blockIdx.y;
  const size_t q_row = static_cast<size_t>(bh) * Nq + blockIdx.x * kTile + r;
  const float* kbase = k + (static_cast<size_t>(bh) * nk_stride + k_off) * kD;
  const float* vbase = v + (static_cast<size_t>(bh) * nk_stride + k_off) * kD;

  if (threadIdx.x == 0) {
    mbar_init(bar, 1);
    fence_mbar_init();
  }
  if (warp == 0) tmem_alloc<512>(tmem_slot);
  split_row_to_smem<kD>(q + q_row * kD, sQ, r);
  fence_proxy_async_smem();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_slot;
  const uint32_t lane_off = static_cast<uint32_t>(warp * 32) << 16;
  const uint32_t q_addr = smem_u32(sQ), kv_addr = smem_u32(sKV);
  constexpr uint32_t idesc_s = make_idesc_bf16(kTile, kTile, 0, 0);     // Q_a (K-major) x K_b^T (K-major)
  constexpr uint32_t idesc_o = make_idesc_bf16(kTile, kD, 0, 1);        // P_a (TMEM) x V_b (MN-major)

  const float scale_log2 = scale * 1.4426950408889634f;
  float m = -CUDART_INF_F, l = 0.f;        // running row max of the scaled scores (log2 domain), running row sum
  uint32_t phase = 0;
  const int n_kv = nk / kTile;
  for (int j = 0; j < n_kv; ++j) {
    // ---- K_j -> shared memory (the P V MMAs of the previous tile have been waited for: the region is free)
    split_row_to_smem<kD>(kbase + (static_cast<size_t>(j) * kTile + r) * kD, sKV, r);
    fence_proxy_async_smem();
    __syncthreads();
    if (threadIdx.x == 0) {
      tc_fence_after();
#pragma unroll
      for (int t = 0; t < 6; ++t) {
        const uint32_t a0 = q_addr + pair_a(t) * Cfg::kTileBytes, b0 = kv_addr + pair_b(t) * Cfg::kTileBytes;
#pragma unroll
        for (int kk = 0; kk < kD / 16; ++kk) {
          const uint32_t off = (kk >> 2) * kPanelBytes + (kk & 3) * 32;
          mma_ss(tmem + tS, make_smem_desc_sw128(a0 + off, 16, 1024), make_smem_desc_sw128(b0 + off, 16, 1024), idesc_s,
                 t > 0 || kk > 0);
        }
      }
      mma_commit(bar);
    }
    mbar_wait(bar, phase);
    phase ^= 1;
    tc_fence_after();
    // ---- V_j -> the same shared memory (S is complete: K_j has been read)
    split_row_to_smem<kD>(vbase + (static_cast<size_t>(j) * kTile + r) * kD, sKV, r);
    fence_proxy_async_smem();
    // ---- online softmax of my row, fp32 (Eq. 2-3)
    float mx = -CUDART_INF_F;
    uint32_t s[kTile];
#pragma unroll
    for (int c = 0; c < 4; ++c) tmem_ld_x32(tmem + tS + lane_off + c * 32, *reinterpret_cast<uint32_t(*)[32]>(&s[c * 32]));
    tmem_wait_ld();
#pragma unroll
    for (int i = 0; i < kTile; ++i) mx = fmaxf(mx, __uint_as_float(s[i]));
    const float m_new = fmaxf(m, mx * scale_log2);
    const float alpha = exp2f(m - m_new);            // 0 on the first tile
    if (j > 0 && __any_sync(0xffffffffu, alpha != 1.0f)) {   // rescale O (the previous P V is complete); warp-uniform:
                                                             // tcgen05.ld / .st are warp-collective
#pragma unroll
      for (int c = 0; c < kD / 32; ++c) {
        uint32_t o[32];
        tmem_ld_x32(tmem + tO + lane_off + c * 32, o);
        tmem_wait_ld();
#pragma unroll
        for (int i = 0; i < 32; ++i) o[i] = __float_as_uint(__uint_as_float(o[i]) * alpha);
        tmem_st_x32(tmem + tO + lane_off + c * 32, o);
      }
    }
    float sum = 0.f;
#pragma unroll
    for (int c = 0; c < 4; ++c) {                    // 32 keys at a time: P -> three bf16 pieces of 16 TMEM columns
      uint32_t ph[16], pm[16], pl[16];
#pragma unroll
      for (int i = 0; i < 32; i += 2) {
        const float p0 = exp2f(fmaf(__uint_as_float(s[c * 32 + i]), scale_log2, -m_new));
        const float p1 = exp2f(fmaf(__uint_as_float(s[c * 32 + i + 1]), scale_log2, -m_new));
        sum += p0 + p1;
        uint16_t h0, m0, l0, h1, m1, l1;
        split3(p0, h0, m0, l0);
        split3(p1, h1, m1, l1);
        ph[i / 2] = static_cast<uint32_t>(h0) | (static_cast<uint32_t>(h1) << 16);
        pm[i / 2] = static_cast<uint32_t>(m0) | (static_cast<uint32_t>(m1) << 16);
        pl[i / 2] = static_cast<uint32_t>(l0) | (static_cast<uint32_t>(l1) << 16);
      }
      tmem_st_x16(tmem + tP + lane_off + c * 16, ph);
      tmem_st_x16(tmem + tP + 64 + lane_off + c * 16, pm);
      tmem_st_x16(tmem + tP + 128 + lane_off + c * 16, pl);
    }
    l = l * alpha + sum;
    m = m_new;
    tmem_wait_st();
    tc_fence_before();
    __syncthreads();
    // ---- O (+)= sum over the six (P_a, V_b) pairs
    if (threadIdx.x == 0) {
      tc_fence_after();
#pragma unroll
      for (int t = 0; t < 6; ++t) {
        const uint32_t b0 = kv_addr + pair_b(t) * Cfg::kTileBytes;
#pragma unroll
        for (int kk = 0; kk < kTile / 16; ++kk)
          mma_ts(tmem + tO, tmem + tP + pair_a(t) * 64 + kk * 8, make_smem_desc_sw128(b0 + kk * 2048, kPanelBytes, 1024),
                 idesc_o, j > 0 || t > 0 || kk > 0);
      }
      mma_commit(bar);
    }
    mbar_wait(bar, phase);
    phase ^= 1;
    tc_fence_after();
  }
  // ---- epilogue: loc_out = O / l, loc_lse = (m + log2 l) ln 2   (natural log of the scaled scores)
  const float inv = 1.0f / l;
  float* orow = o_out + q_row * kD;
#pragma unroll
  for (int c = 0; c < kD / 32; ++c) {
    uint32_t o[32];
    tmem_ld_x32(tmem + tO + lane_off + c * 32, o);
    tmem_wait_ld();
#pragma unroll
    for (int i = 0; i < 32; i += 4)
      *reinterpret_cast<float4*>(orow + c * 32 + i) =
          make_float4(__uint_as_float(o[i]) * inv, __uint_as_float(o[i + 1]) * inv, __uint_as_float(o[i + 2]) * inv,
                      __uint_as_float(o[i + 3]) * inv);
  }
  lse_out[q_row] = (m + log2f(l)) * 0.6931471805599453f;
  tc_fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc<512>(tmem);
}

template <int kD>
cudaError_t launch_t(const float* q, const float* k, const float* v, float* o_out, float* lse_out, int BH, int Nq,
                     int nk_stride, int k_off, int nk, float scale, cudaStream_t stream) {
  using Cfg = SplitCfg<kD>;
  auto kern = attn_chunk_f32_split_kernel<kD>;
  static unsigned char configured[kMaxDevices];
  if (cudaError_t e = set_max_dyn_smem_once(kern, Cfg::kSmemBytes, configured); e != cudaSuccess) return e;
  dim3 grid(Nq / kTile, BH);
  kern<<<grid, kTile, Cfg::kSmemBytes, stream>>>(q, k, v, o_out, lse_out, Nq, nk_stride, k_off, nk, scale);
  count_launch();
  return cudaGetLastError();
}

}  // namespace

cudaError_t launch_attn_chunk_f32(const float* q, const float* k, const float* v, float* o_out, float* lse_out, int BH,
                                  int Nq, int nk_stride, int k_off, int nk, int d, float scale, cudaStream_t stream) {
  if (d == 64) return launch_t<64>(q, k, v, o_out, lse_out, BH, Nq, nk_stride, k_off, nk, scale, stream);
  return launch_t<128>(q, k, v, o_out, lse_out, BH, Nq, nk_stride, k_off, nk, scale, stream);
}

}  // namespace ringx
