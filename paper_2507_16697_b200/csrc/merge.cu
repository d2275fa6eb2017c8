// merge.cu -- HBM-bound helper kernels of the RingX hot path:
//   lse_merge_kernel   two-operand Eq. (5): SURVEY.md §8(a) row a5/a6
//   bwd_preprocess     D_i = sum_c dO_ic O_ic, lse2_i = LSE_i log2(e), zeroing of the fp32 dQ accumulator: row a7
//   dq_convert         dq = bf16(scale * dq_acc): row a9
//   eq5_scale / eq5_finalize   Eq. (5) in its N-operand form (num, den before / after the cross-device sums;
//                      PAPER.md:137-143): the RingX_a merge, SURVEY.md §8(f) NEXT-1
// Roofline: HBM bandwidth.  Algorithmic bytes per row: merge 2*(d*e_in+4) read + (d*e_out+4)
// written; preprocess 2*d*2 read + 4 written (+ d*4 zeroed); convert d*4 read + d*2 written.
#include "kernels.cuh"

namespace ringx {

namespace {

constexpr int kMergeThreads = 256;
constexpr int kRowUnroll = 4;

template <typename T>
struct Vec4;  // 4 consecutive elements of a row
template <>
struct Vec4<float> {
  static __device__ __forceinline__ float4 load(const void* p, size_t i4) {
    return __ldcs(reinterpret_cast<const float4*>(p) + i4);
  }
  static __device__ __forceinline__ void store(void* p, size_t i4, float4 v) {
    __stcs(reinterpret_cast<float4*>(p) + i4, v);
  }
};
template <>
struct Vec4<__nv_bfloat16> {
  static __device__ __forceinline__ float4 load(const void* p, size_t i4) {
    uint2 u = __ldcs(reinterpret_cast<const uint2*>(p) + i4);
    float4 v;
    v.x = __uint_as_float(u.x << 16);
    v.y = __uint_as_float(u.x & 0xFFFF0000u);
    v.z = __uint_as_float(u.y << 16);
    v.w = __uint_as_float(u.y & 0xFFFF0000u);
    return v;
  }
  static __device__ __forceinline__ void store(void* p, size_t i4, float4 v) {
    uint2 u;
    u.x = ptx::pack_bf16x2(v.x, v.y);
    u.y = ptx::pack_bf16x2(v.z, v.w);
    __stcs(reinterpret_cast<uint2*>(p) + i4, u);
  }
};

// Weights of the two-operand Eq. (5).  -inf operands get weight 0 (reading g12).
__device__ __forceinline__ void merge_weights(float la, float lb, float& wa, float& wb, float& lse) {
  const float m = fmaxf(la, lb);
  if (m == -INFINITY) {
    wa = 0.f; wb = 0.f; lse = -INFINITY;
    return;
  }
  const float ea = expf(la - m), eb = expf(lb - m);   // exp(-inf) = 0; NaN propagates
  const float den = ea + eb;
  const float inv = 1.0f / den;
  wa = ea * inv;
  wb = eb * inv;
  lse = m + logf(den);
}

// One group of kLanes lanes owns a row (d/4 = kLanes * iters vectors).  A warp owns 32/kLanes rows
// per step and kRowUnroll steps are in flight, so the lse read, the two o reads and the write of a
// row all come from one warp: running in place on operand a is race-free.
template <typename TIn, typename TOut, int kLanes>
__global__ void __launch_bounds__(kMergeThreads)
lse_merge_kernel(const void* o_a, const float* lse_a, const void* __restrict__ o_b,
                 const float* __restrict__ lse_b, void* o_out, float* lse_out, long long rows, int d) {
  // o_a / lse_a carry no __restrict__: the header lets o_out alias o_a and lse_out alias lse_a (in-place merge)
  constexpr int kRowsPerWarp = 32 / kLanes;
  const int lane = threadIdx.x & 31;
  const int sub = lane / kLanes, l = lane % kLanes;
  const int vecs = d >> 2;
  const long long warp_global = (long long)blockIdx.x * (kMergeThreads / 32) + (threadIdx.x >> 5);
  const long long warp_count = (long long)gridDim.x * (kMergeThreads / 32);
  const long long rows_per_iter = (long long)kRowsPerWarp * kRowUnroll;
  for (long long base = warp_global * rows_per_iter; base < rows; base += warp_count * rows_per_iter) {
    float wa[kRowUnroll], wb[kRowUnroll], lse[kRowUnroll];
    long long row[kRowUnroll];
#pragma unroll
    for (int u = 0; u < kRowUnroll; ++u) {
      row[u] = base + u * kRowsPerWarp + sub;
      float la = -INFINITY, lb = -INFINITY;
      if (row[u] < rows) {
        la = lse_a[row[u]];
        lb = lse_b[row[u]];
      }
      merge_weights(la, lb, wa[u], wb[u], lse[u]);
    }
    for (int v0 = 0; v0 < vecs; v0 += kLanes) {
      const int v = v0 + l;
      float4 a[kRowUnroll], b[kRowUnroll];
#pragma unroll
      for (int u = 0; u < kRowUnroll; ++u)
        if (row[u] < rows && v < vecs) {
          a[u] = Vec4<TIn>::load(o_a, (size_t)row[u] * vecs + v);
          b[u] = Vec4<TIn>::load(o_b, (size_t)row[u] * vecs + v);
        }
#pragma unroll
      for (int u = 0; u < kRowUnroll; ++u)
        if (row[u] < rows && v < vecs) {
          float4 r;
          // weight-0 operands are skipped so that garbage (even NaN) behind an empty chunk is ignored
          r.x = (wa[u] != 0.f ? wa[u] * a[u].x : 0.f) + (wb[u] != 0.f ? wb[u] * b[u].x : 0.f);
          r.y = (wa[u] != 0.f ? wa[u] * a[u].y : 0.f) + (wb[u] != 0.f ? wb[u] * b[u].y : 0.f);
          r.z = (wa[u] != 0.f ? wa[u] * a[u].z : 0.f) + (wb[u] != 0.f ? wb[u] * b[u].z : 0.f);
          r.w = (wa[u] != 0.f ? wa[u] * a[u].w : 0.f) + (wb[u] != 0.f ? wb[u] * b[u].w : 0.f);
          Vec4<TOut>::store(o_out, (size_t)row[u] * vecs + v, r);
        }
    }
    __syncwarp();   // every lane has read lse_a of its rows before lane 0 of the group overwrites it
#pragma unroll
    for (int u = 0; u < kRowUnroll; ++u)
      if (row[u] < rows && l == 0) lse_out[row[u]] = lse[u];
  }
}

template <typename TIn, typename TOut>
cudaError_t launch_merge_t(const void* o_a, const float* lse_a, const void* o_b, const float* lse_b, void* o_out,
                           float* lse_out, long long rows, int d, cudaStream_t stream) {
  const int vecs = d / 4;
  int lanes = 32;
  if (vecs < 32 && (vecs & (vecs - 1)) == 0) lanes = vecs;
  const long long rows_per_block = (long long)(kMergeThreads / 32) * (32 / lanes) * kRowUnroll;
  long long blocks = (rows + rows_per_block - 1) / rows_per_block;
  const long long max_blocks = (long long)sm_count() * 8 * 4;   // 8 CTAs of 256 threads per SM, 4 waves
  if (blocks > max_blocks) blocks = max_blocks;
  if (blocks < 1) blocks = 1;
#define RINGX_MERGE_CASE(L)                                                                                     \
  case L:                                                                                                       \
    lse_merge_kernel<TIn, TOut, L><<<(unsigned)blocks, kMergeThreads, 0, stream>>>(o_a, lse_a, o_b, lse_b, o_out, \
                                                                                   lse_out, rows, d);           \
    break;
  switch (lanes) {
    RINGX_MERGE_CASE(2)
    RINGX_MERGE_CASE(4)
    RINGX_MERGE_CASE(8)
    RINGX_MERGE_CASE(16)
    default:
      lse_merge_kernel<TIn, TOut, 32><<<(unsigned)blocks, kMergeThreads, 0, stream>>>(o_a, lse_a, o_b, lse_b, o_out,
                                                                                      lse_out, rows, d);
  }
#undef RINGX_MERGE_CASE
  return cudaGetLastError();
}

// ---------------------------------------------------------------- Eq. 5, N-operand form (RingX_a: PAPER.md:137-143)
// One operand's share before the cross-device sums: w = exp(loc_lse - lse_max), num = w * loc_out, den = w.
// lse_max is the all-reduce(max) of loc_lse over the devices; an operand with loc_lse = -inf (or a row whose
// lse_max is -inf) contributes 0 and its loc_out is not read into the result.  One thread per float4.
__global__ void __launch_bounds__(256)
eq5_scale_kernel(const float4* loc_out, const float* __restrict__ loc_lse,     // num may alias loc_out (in place):
                 const float* __restrict__ lse_max, float4* num, float* __restrict__ den, long long rows,   // no restrict
                 int vecs) {
  const long long total = rows * vecs, stride = (long long)gridDim.x * blockDim.x;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += stride) {
    const long long r = i / vecs;
    const float l = loc_lse[r], m = lse_max[r];
    const float w = (l == -INFINITY || m == -INFINITY) ? 0.f : expf(l - m);
    float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
    if (w != 0.f) {
      v = __ldcs(loc_out + i);
      v.x *= w; v.y *= w; v.z *= w; v.w *= w;
    }
    __stcs(num + i, v);
    if (i - r * vecs == 0) den[r] = w;
  }
}

// After the sums: o = num / den, lse = lse_max + ln(den); den = 0 (every operand empty) gives o = 0, lse = -inf.
template <typename TOut>
__global__ void __launch_bounds__(256)
eq5_finalize_kernel(const float4* num, const float* __restrict__ den, const float* lse_max,   // o_out may alias num and
                    void* o_out, float* lse_out, long long rows, int vecs) {                  // lse_out lse_max: no restrict
  const long long total = rows * vecs, stride = (long long)gridDim.x * blockDim.x;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += stride) {
    const long long r = i / vecs;
    const float dn = den[r];
    float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
    if (dn != 0.f) {
      const float inv = 1.0f / dn;
      v = __ldcs(num + i);
      v.x *= inv; v.y *= inv; v.z *= inv; v.w *= inv;
    }
    Vec4<TOut>::store(o_out, (size_t)i, v);
    if (i - r * vecs == 0) lse_out[r] = dn != 0.f ? lse_max[r] + logf(dn) : -INFINITY;   // NaN den propagates
  }
}

// Eq. 5 over the s key splits of one chunk pass (split-KV), optionally with the running (o_acc, lse_acc) as one more
// operand: parts [s][rows,d] fp32, lses [s][rows].  One thread per float4; s <= kMaxSplits so the weights sit in
// registers.  An operand with lse = -inf has weight 0; every operand empty gives o = 0, lse = -inf.
constexpr int kMaxSplits = 8;
template <typename TOut>
__global__ void __launch_bounds__(256)
split_merge_kernel(const float4* __restrict__ parts, const float* __restrict__ lses, long long part_stride_vecs,
                   long long rows, int s, const float4* o_acc, const float* __restrict__ lse_acc,   // o_out may alias
                   void* o_out, float* __restrict__ lse_out, int vecs) {                           // o_acc: no restrict
  const long long total = rows * vecs, stride = (long long)gridDim.x * blockDim.x;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += stride) {
    const long long r = i / vecs;
    float l[kMaxSplits + 1];
    float m = -INFINITY;
#pragma unroll
    for (int p = 0; p < kMaxSplits; ++p) {
      l[p] = p < s ? lses[p * rows + r] : -INFINITY;
      m = fmaxf(m, l[p]);
    }
    l[kMaxSplits] = lse_acc ? lse_acc[r] : -INFINITY;
    m = fmaxf(m, l[kMaxSplits]);
    const float ms = (m == -INFINITY) ? 0.f : m;
    float den = 0.f;
    float4 num = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
    for (int p = 0; p <= kMaxSplits; ++p) {
      if (l[p] == -INFINITY && !(l[p] != l[p])) continue;            // empty operand: weight 0, data not read
      const float w = __expf(l[p] - ms);
      const float4 v = p < kMaxSplits ? __ldcs(parts + p * part_stride_vecs + i) : __ldcs(o_acc + i);
      den += w;
      num.x = fmaf(w, v.x, num.x); num.y = fmaf(w, v.y, num.y); num.z = fmaf(w, v.z, num.z); num.w = fmaf(w, v.w, num.w);
    }
    float4 o = make_float4(0.f, 0.f, 0.f, 0.f);
    if (den != 0.f) {
      const float inv = 1.0f / den;
      o = make_float4(num.x * inv, num.y * inv, num.z * inv, num.w * inv);
    }
    Vec4<TOut>::store(o_out, (size_t)i, o);
    if (i - r * vecs == 0) lse_out[r] = den != 0.f ? ms + logf(den) : -INFINITY;
  }
}

// ---------------------------------------------------------------- backward helpers
// D_i = sum_c dO_ic * O_ic (fp32), one 16-lane (d=64: 8 B/lane... ) group per row: each lane takes
// 8 bf16 (16 B) of dO and of O; d/8 lanes per row.  Stores scale * D_i; zeroes the row of the fp32 dQ accumulator
// when zero_dq.
template <int kLanes>
__global__ void __launch_bounds__(256)
bwd_preprocess_kernel(const uint4* __restrict__ o, const uint4* __restrict__ dO, const float* __restrict__ lse,
                      float* __restrict__ D, float* __restrict__ lse2, float4* __restrict__ dq_acc, long long rows,
                      float scale, bool zero_dq, long long rows_per_head, long long n_stat) {
  constexpr int kRowsPerWarp = 32 / kLanes;
  const int lane = threadIdx.x & 31, sub = lane / kLanes, l = lane % kLanes;
  const long long warp_global = (long long)blockIdx.x * 8 + (threadIdx.x >> 5);
  const long long warp_count = (long long)gridDim.x * 8;
  for (long long base = warp_global * kRowsPerWarp * 4; base < rows; base += warp_count * kRowsPerWarp * 4) {
    uint4 a[4], b[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const long long r = base + u * kRowsPerWarp + sub;
      if (r < rows) {
        a[u] = __ldg(o + r * kLanes + l);
        b[u] = __ldg(dO + r * kLanes + l);
      }
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const long long r = base + u * kRowsPerWarp + sub;
      float s = 0.f;
      if (r < rows) {
        const uint32_t* pa = reinterpret_cast<const uint32_t*>(&a[u]);
        const uint32_t* pb = reinterpret_cast<const uint32_t*>(&b[u]);
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          s = fmaf(__uint_as_float(pa[i] << 16), __uint_as_float(pb[i] << 16), s);
          s = fmaf(__uint_as_float(pa[i] & 0xFFFF0000u), __uint_as_float(pb[i] & 0xFFFF0000u), s);
        }
        if (zero_dq) {
          const float4 z = make_float4(0.f, 0.f, 0.f, 0.f);
          dq_acc[(r * kLanes + l) * 2] = z;
          dq_acc[(r * kLanes + l) * 2 + 1] = z;
        }
      }
#pragma unroll
      for (int off = kLanes / 2; off > 0; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
      if (r < rows && l == 0) {
        // D, lse2 are [heads][n_stat]: n_stat = rows_per_head rounded up to the 128-row tile (equal unless the sequence
        // is ragged), so that the backward kernel's 128-entry loads of a head's last tile stay inside the head
        const long long rs = n_stat == rows_per_head ? r : (r / rows_per_head) * n_stat + r % rows_per_head;
        D[rs] = s * scale;                         // phase B of the backward forms scale*dP - scale*D
        lse2[rs] = lse[r] * 1.4426950408889634f;  // the backward kernel works in the exp2 domain
      }
    }
  }
}

// the padding of a ragged head in D, lse2: lse2 = +inf makes P = exp2(x - lse2) = 0 for query rows that do not exist
__global__ void __launch_bounds__(128)
bwd_stat_pad_kernel(float* __restrict__ D, float* __restrict__ lse2, int rows_per_head, int n_stat) {
  const int n = rows_per_head + threadIdx.x;
  if (n < n_stat) {
    D[(long long)blockIdx.x * n_stat + n] = 0.f;
    lse2[(long long)blockIdx.x * n_stat + n] = CUDART_INF_F;
  }
}

__global__ void __launch_bounds__(256)
dq_convert_kernel(const float4* __restrict__ dq_acc, uint2* __restrict__ dq, long long n4, float scale) {
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += stride) {
    const float4 v = __ldcs(dq_acc + i);
    uint2 u;
    u.x = ptx::pack_bf16x2(v.x * scale, v.y * scale);
    u.y = ptx::pack_bf16x2(v.z * scale, v.w * scale);
    dq[i] = u;
  }
}

// ---------------------------------------------------------------- deterministic dQ: int32 fixed-point accumulator
// (ringx_set_deterministic).  Integer adds are associative, so TMA reduce-adds of integers give the same sum in any
// arrival order.  Row r gets a scale qs[r] with |dQ_rc| * qs[r] <= 1.5e9 < 2^31 guaranteed by
//   |dQ_rc| = scale |sum_j P_rj (dP_rj - D_r) K_jc| <= scale (sum_j P_rj) (max_j|dO_r.V_j| + |D_r|) max_j|K_jc|
//                                                 <= scale (||dO_r|| max_j||V_j|| + |D_r|) max_jc|K_jc|
// over the keys j of THIS call, with sum_j P_rj <= 1 because P is formed from the LSE over all keys of the sequence.
// |D_r| is read from the preprocess buffer, not bounded by ||dO_r|| max||V||: in a per-device step (ringx_attn_bwd_partial)
// O, and with it D_r = dO_r.O_r, comes from the keys of ALL devices, whose values may be far larger than this step's (or
// this step's V may be all zeros) -- D_r then lies outside the hull of the local dP_rj.
// (the partial sums may wrap: two's-complement adds are exact modulo 2^32, only the final value has to fit).
// Non-finite inputs: a NaN/Inf in dO_r or O_r (through D_r) or in the K, V of the call makes the bound non-finite; qs[r] is
// then NaN and the row of dq comes out NaN, as the fp32 accumulator would give (a non-finite Q or lse is NOT detected: the
// kernel's fp32 contribution is NaN and rounds to integer 0).

// kvmax[2h] = max_j ||V_j||^2, kvmax[2h+1] = max_jc |K_jc| over the nk key rows [k_off, k_off+nk) of kv head h
// (atomicMax on the bit patterns of non-negative floats: order-independent).  grid = (blocks, BH); kvmax zeroed before.
// V rows are kLanesV uint4 wide (d_v = 8 kLanesV), K rows k_vecs uint4 wide (any width: only max |.| is needed).
template <int kLanesV>
__global__ void __launch_bounds__(256)
kv_absmax_kernel(const uint4* __restrict__ k, const uint4* __restrict__ v, unsigned* __restrict__ kvmax, int nk_stride,
                 int k_off, int nk, int k_vecs) {
  constexpr int kRowsPerWarp = 32 / kLanesV;
  const int lane = threadIdx.x & 31, sub = lane / kLanesV, l = lane % kLanesV;
  const int bh = blockIdx.y;
  const long long head0 = (long long)bh * nk_stride + k_off;
  float vmax2 = 0.f, kmax = 0.f;
  for (int base = (blockIdx.x * 8 + (threadIdx.x >> 5)) * kRowsPerWarp; base < nk; base += gridDim.x * 8 * kRowsPerWarp) {
    const int r = base + sub;
    uint4 b = make_uint4(0u, 0u, 0u, 0u);
    if (r < nk) b = __ldg(v + (head0 + r) * kLanesV + l);
    const uint32_t* pb = reinterpret_cast<const uint32_t*>(&b);
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const float v0 = __uint_as_float(pb[i] << 16), v1 = __uint_as_float(pb[i] & 0xFFFF0000u);
      s = fmaf(v0, v0, s);
      s = fmaf(v1, v1, s);
    }
#pragma unroll
    for (int off = kLanesV / 2; off > 0; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
    vmax2 = s != s ? CUDART_INF_F : fmaxf(vmax2, s);      // fmaxf drops a NaN: keep it as +inf (the bound turns non-finite)
  }
  const uint4* kh = k + head0 * k_vecs;
  for (long long i = (long long)blockIdx.x * 256 + threadIdx.x; i < (long long)nk * k_vecs; i += (long long)gridDim.x * 256) {
    const uint4 a = __ldg(kh + i);
    const uint32_t* pa = reinterpret_cast<const uint32_t*>(&a);
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const float k0 = fabsf(__uint_as_float(pa[j] << 16)), k1 = fabsf(__uint_as_float(pa[j] & 0xFFFF0000u));
      kmax = (k0 != k0 || k1 != k1) ? CUDART_INF_F : fmaxf(kmax, fmaxf(k0, k1));
    }
  }
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) {
    vmax2 = fmaxf(vmax2, __shfl_xor_sync(0xffffffffu, vmax2, off));
    kmax = fmaxf(kmax, __shfl_xor_sync(0xffffffffu, kmax, off));
  }
  if (lane == 0) {
    atomicMax(kvmax + 2 * bh, __float_as_uint(vmax2));
    atomicMax(kvmax + 2 * bh + 1, __float_as_uint(kmax));
  }
}

// qs[r] = 1.5e9 / bound_r (clamped to [2^-100, 2^100]; NaN when bound_r is not finite),
// bound_r = 1.015625 * (scale * ||dO_r|| * sqrt(kvmax[2h]) + |Ds_r|) * kvmax[2h+1], h = r / rows_per_head, where
// Ds = scale * D is launch_bwd_preprocess's buffer ([heads][n_stat] layout) -- the very values the backward kernel subtracts.
// The 1.015625 covers the bf16 rounding of dS and a row sum of P up to 1.001; 1.5e9 + one rounding of 1/2 per key tile
// stays below 2^31.
template <int kLanes>
__global__ void __launch_bounds__(256)
dq_fixed_scale_kernel(const uint4* __restrict__ dO, const float* __restrict__ kvmax, const float* __restrict__ Ds,
                      float* __restrict__ qs, long long rows, long long rows_per_head, long long n_stat, float scale) {
  constexpr int kRowsPerWarp = 32 / kLanes;
  const int lane = threadIdx.x & 31, sub = lane / kLanes, l = lane % kLanes;
  const long long warp_global = (long long)blockIdx.x * 8 + (threadIdx.x >> 5);
  const long long warp_count = (long long)gridDim.x * 8;
  for (long long base = warp_global * kRowsPerWarp; base < rows; base += warp_count * kRowsPerWarp) {
    const long long r = base + sub;
    float s = 0.f;
    if (r < rows) {
      const uint4 b = __ldg(dO + r * kLanes + l);
      const uint32_t* pb = reinterpret_cast<const uint32_t*>(&b);
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const float v0 = __uint_as_float(pb[i] << 16), v1 = __uint_as_float(pb[i] & 0xFFFF0000u);
        s = fmaf(v0, v0, s);
        s = fmaf(v1, v1, s);
      }
    }
#pragma unroll
    for (int off = kLanes / 2; off > 0; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
    if (r < rows && l == 0) {
      const long long h = r / rows_per_head;
      const float ds = fabsf(__ldg(Ds + h * n_stat + (r - h * rows_per_head)));
      const float bound = 1.015625f * (scale * sqrtf(s) * sqrtf(kvmax[2 * h]) + ds) * kvmax[2 * h + 1];
      const float q = fminf(fmaxf(1.5e9f / fmaxf(bound, 1e-37f), 7.8886e-31f), 1.2676506e30f);
      qs[r] = bound <= 3.0e38f ? q : CUDART_NAN_F;          // NaN or Inf bound: the row of dq is NaN, not silently finite
    }
  }
}

// dq (bf16) = dq_fix / qs[row], vecs = d / 4 int4 per row
__global__ void __launch_bounds__(256)
dq_fixed_convert_kernel(const int4* __restrict__ dq_fix, const float* __restrict__ qs, uint2* __restrict__ dq,
                        long long n4, int vecs) {
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += stride) {
    const int4 v = __ldcs(dq_fix + i);
    const float inv = 1.0f / __ldg(qs + i / vecs);
    uint2 u;
    u.x = ptx::pack_bf16x2(static_cast<float>(v.x) * inv, static_cast<float>(v.y) * inv);
    u.y = ptx::pack_bf16x2(static_cast<float>(v.z) * inv, static_cast<float>(v.w) * inv);
    dq[i] = u;
  }
}

// dq_acc (fp32, the caller's accumulator across the steps of a RingX backward) += dq_fix / qs[row]
__global__ void __launch_bounds__(256)
dq_fixed_accumulate_kernel(const int4* __restrict__ dq_fix, const float* __restrict__ qs, float4* __restrict__ dq_acc,
                           long long n4, int vecs) {
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += stride) {
    const int4 v = __ldcs(dq_fix + i);
    const float inv = 1.0f / __ldg(qs + i / vecs);
    float4 a = dq_acc[i];
    a.x += static_cast<float>(v.x) * inv;
    a.y += static_cast<float>(v.y) * inv;
    a.z += static_cast<float>(v.z) * inv;
    a.w += static_cast<float>(v.w) * inv;
    dq_acc[i] = a;
  }
}

}  // namespace

cudaError_t launch_lse_merge(const void* o_a, const float* lse_a, const void* o_b, const float* lse_b, void* o_out,
                             float* lse_out, long long rows, int d, int in_dtype, int out_dtype,
                             cudaStream_t stream) {
  if (rows == 0) return cudaSuccess;
  if (in_dtype == RINGX_F32 && out_dtype == RINGX_F32)
    return launch_merge_t<float, float>(o_a, lse_a, o_b, lse_b, o_out, lse_out, rows, d, stream);
  if (in_dtype == RINGX_F32 && out_dtype == RINGX_BF16)
    return launch_merge_t<float, __nv_bfloat16>(o_a, lse_a, o_b, lse_b, o_out, lse_out, rows, d, stream);
  if (in_dtype == RINGX_BF16 && out_dtype == RINGX_F32)
    return launch_merge_t<__nv_bfloat16, float>(o_a, lse_a, o_b, lse_b, o_out, lse_out, rows, d, stream);
  return launch_merge_t<__nv_bfloat16, __nv_bfloat16>(o_a, lse_a, o_b, lse_b, o_out, lse_out, rows, d, stream);
}

static unsigned eq5_blocks(long long total) {
  long long blocks = (total + 255) / 256;
  if (blocks > (long long)sm_count() * 8 * 4) blocks = (long long)sm_count() * 8 * 4;
  return (unsigned)(blocks < 1 ? 1 : blocks);
}

cudaError_t launch_eq5_scale(const float* loc_out, const float* loc_lse, const float* lse_max, float* num, float* den,
                             long long rows, int d, cudaStream_t stream) {
  if (rows == 0) return cudaSuccess;
  eq5_scale_kernel<<<eq5_blocks(rows * (d / 4)), 256, 0, stream>>>((const float4*)loc_out, loc_lse, lse_max,
                                                                  (float4*)num, den, rows, d / 4);
  return cudaGetLastError();
}

cudaError_t launch_eq5_finalize(const float* num, const float* den, const float* lse_max, void* o_out, float* lse_out,
                                long long rows, int d, int out_dtype, cudaStream_t stream) {
  if (rows == 0) return cudaSuccess;
  if (out_dtype == RINGX_BF16)
    eq5_finalize_kernel<__nv_bfloat16><<<eq5_blocks(rows * (d / 4)), 256, 0, stream>>>(
        (const float4*)num, den, lse_max, o_out, lse_out, rows, d / 4);
  else
    eq5_finalize_kernel<float><<<eq5_blocks(rows * (d / 4)), 256, 0, stream>>>((const float4*)num, den, lse_max, o_out,
                                                                                lse_out, rows, d / 4);
  return cudaGetLastError();
}

cudaError_t launch_split_merge(const float* parts, const float* lses, long long rows, int d, int splits,
                               const float* o_acc, const float* lse_acc, void* o_out, float* lse_out, int out_dtype,
                               cudaStream_t stream) {
  if (rows == 0) return cudaSuccess;
  if (splits < 1 || splits > kMaxSplits) return cudaErrorInvalidValue;
  const int vecs = d / 4;
  if (out_dtype == RINGX_BF16)
    split_merge_kernel<__nv_bfloat16><<<eq5_blocks(rows * vecs), 256, 0, stream>>>(
        (const float4*)parts, lses, rows * vecs, rows, splits, (const float4*)o_acc, lse_acc, o_out, lse_out, vecs);
  else
    split_merge_kernel<float><<<eq5_blocks(rows * vecs), 256, 0, stream>>>(
        (const float4*)parts, lses, rows * vecs, rows, splits, (const float4*)o_acc, lse_acc, o_out, lse_out, vecs);
  return cudaGetLastError();
}

cudaError_t launch_bwd_preprocess(const void* o, const void* dO, const float* lse, float* D, float* lse2,
                                  float* dq_acc, long long rows, int d, float scale, bool zero_dq,
                                  cudaStream_t stream, long long rows_per_head) {
  const long long n_stat = rows_per_head <= 0 ? rows : (rows_per_head + 127) / 128 * 128;
  if (rows_per_head <= 0) rows_per_head = rows;
  if (n_stat != rows_per_head)
    bwd_stat_pad_kernel<<<(unsigned)(rows / rows_per_head), 128, 0, stream>>>(D, lse2, (int)rows_per_head, (int)n_stat);
  const int lanes = d / 8;   // 8 or 16
  const long long rows_per_block = 8LL * (32 / lanes) * 4;
  long long blocks = (rows + rows_per_block - 1) / rows_per_block;
  if (blocks > (long long)sm_count() * 8 * 4) blocks = (long long)sm_count() * 8 * 4;
  if (lanes == 8)
    bwd_preprocess_kernel<8><<<(unsigned)blocks, 256, 0, stream>>>((const uint4*)o, (const uint4*)dO, lse, D, lse2,
                                                                   (float4*)dq_acc, rows, scale, zero_dq, rows_per_head, n_stat);
  else
    bwd_preprocess_kernel<16><<<(unsigned)blocks, 256, 0, stream>>>((const uint4*)o, (const uint4*)dO, lse, D, lse2,
                                                                    (float4*)dq_acc, rows, scale, zero_dq, rows_per_head, n_stat);
  return cudaGetLastError();
}

cudaError_t launch_dq_convert(const float* dq_acc, void* dq, long long n, float scale, cudaStream_t stream) {
  const long long n4 = n / 4;
  long long blocks = (n4 + 255) / 256;
  if (blocks > (long long)sm_count() * 8 * 4) blocks = (long long)sm_count() * 8 * 4;
  dq_convert_kernel<<<(unsigned)blocks, 256, 0, stream>>>((const float4*)dq_acc, (uint2*)dq, n4, scale);
  return cudaGetLastError();
}

cudaError_t launch_dq_fixed_scale(const void* k, const void* v, const void* dO, const float* Ds, float* kvmax, float* qs,
                                  int BH, long long rows_per_head, int nk_stride, int k_off, int nk, int d_k, int d_v,
                                  float scale, cudaStream_t stream) {
  cudaError_t e = cudaMemsetAsync(kvmax, 0, (size_t)BH * 2 * sizeof(float), stream);
  if (e != cudaSuccess) return e;
  const int lanes = d_v / 8;   // 8 or 16: V rows and dO rows
  const int rows_per_block = 8 * (32 / lanes);
  int bx = (nk + rows_per_block - 1) / rows_per_block;
  const int cap = (sm_count() * 8 + BH - 1) / BH;
  if (bx > cap) bx = cap;
  const dim3 grid((unsigned)bx, (unsigned)BH);
  const long long rows = (long long)BH * rows_per_head;
  const long long n_stat = (rows_per_head + 127) / 128 * 128;      // launch_bwd_preprocess's per-head pitch of D
  long long blocks = (rows + rows_per_block - 1) / rows_per_block;
  if (blocks > (long long)sm_count() * 8 * 4) blocks = (long long)sm_count() * 8 * 4;
  if (lanes == 8) {
    kv_absmax_kernel<8><<<grid, 256, 0, stream>>>((const uint4*)k, (const uint4*)v, (unsigned*)kvmax, nk_stride, k_off, nk, d_k / 8);
    dq_fixed_scale_kernel<8><<<(unsigned)blocks, 256, 0, stream>>>((const uint4*)dO, kvmax, Ds, qs, rows, rows_per_head, n_stat, scale);
  } else {
    kv_absmax_kernel<16><<<grid, 256, 0, stream>>>((const uint4*)k, (const uint4*)v, (unsigned*)kvmax, nk_stride, k_off, nk, d_k / 8);
    dq_fixed_scale_kernel<16><<<(unsigned)blocks, 256, 0, stream>>>((const uint4*)dO, kvmax, Ds, qs, rows, rows_per_head, n_stat, scale);
  }
  return cudaGetLastError();
}

cudaError_t launch_dq_fixed_finish(const int* dq_fix, const float* qs, void* dq_bf16, float* dq_acc, long long rows, int d,
                                   cudaStream_t stream) {
  const long long n4 = rows * d / 4;
  long long blocks = (n4 + 255) / 256;
  if (blocks > (long long)sm_count() * 8 * 4) blocks = (long long)sm_count() * 8 * 4;
  if (dq_bf16)
    dq_fixed_convert_kernel<<<(unsigned)blocks, 256, 0, stream>>>((const int4*)dq_fix, qs, (uint2*)dq_bf16, n4, d / 4);
  else
    dq_fixed_accumulate_kernel<<<(unsigned)blocks, 256, 0, stream>>>((const int4*)dq_fix, qs, (float4*)dq_acc, n4, d / 4);
  return cudaGetLastError();
}

}  // namespace ringx
