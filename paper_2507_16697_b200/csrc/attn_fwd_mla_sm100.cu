// attn_fwd_mla_sm100.cu -- one KV-chunk pass of the forward for multi-head LATENT attention shapes (SURVEY.md §8(f)
// NEXT-3; the paper names MHA / GQA / MLA as the layer designs RingX is compatible with): in its
// materialised form an MLA layer attends with d_qk = 192 (128 "nope" + 64 rotary dimensions) and d_v = 128, i.e. the
// same Eq. 1 / Eq. 5 with a score contraction that is longer than the value width:
//   loc_out = softmax(scale q K_c^T) V_c,  loc_lse = log sum_j exp(scale q.k_j),   q, k in R^192, v in R^128.
//
// The d = 128 kernel's structure (attn_fwd_sm100.cu: two 128-row query tiles ping-pong through S_0 S_1 O_0 O_1 in TMEM,
// thread = query row, lazy running max, P handed over in two 64-key halves), with what d_qk != d_v changes:
//   * S_t = Q_t K_j^T runs 12 K-steps over three 64-column panels; O_t += P_t V_j is unchanged (N = 128).  TMEM is the
//     same 2 x 128 + 2 x 128 columns.
//   * Shared memory is the constraint: two Q tiles of 192 columns are 96 KB, a K tile 48 KB, a V tile 32 KB.  One ring
//     of equal slots would hold two tiles; instead K and V have rings of their own -- K: 2 slots of 48 KB; V: 2 slots of
//     HALF a tile (64 keys x 128 = 16 KB), because O += P V is issued in two 64-key halves anyway: half h of V_{j+1}
//     can land as soon as tile 1's half-h MMAs of step j are done, 256 clocks before the whole V_j is free.
//     96 + 96 + 32 KB = 224 KB.
//   * one CTA per work item (256 query rows of one head); items here are long (d_qk = 192 layers run at C3-like
//     lengths), so the persistent scheduler of the d = 64 / 128 kernel would buy nothing.
// Roles (384 threads; setmaxnreg 224 / 56): warps 0-3 / 4-7 softmax warpgroups of query tile 0 / 1, warp 8 TMA producer,
// warp 9 MMA issuer, warps 10-11 idle.
#include "kernels.cuh"

namespace ringx {
namespace {

using namespace ptx;

constexpr int kBlockM = 128, kBlockN = 128;
constexpr int kDqk = 192, kDv = 128;
constexpr float kRescaleThreshold = 8.0f;   // log2 units
constexpr int kPanelBytes = 128 * 128;                      // 128 rows x 128 B (64 bf16)
constexpr int kQkTileBytes = (kDqk / 64) * kPanelBytes;     // 48 KB
constexpr int kVHalfPanelBytes = 64 * 128;                  // 64 keys x 128 B
constexpr int kVHalfBytes = (kDv / 64) * kVHalfPanelBytes;  // 16 KB: 64 keys x 128 columns
constexpr int kKStages = 2;
constexpr int kThreads = 384;
constexpr int kSoftmaxRegs = 224, kAuxRegs = 56;
constexpr int kBarBytes = 256;
constexpr int kSmemBytes = 1024 + 2 * kQkTileBytes + kKStages * kQkTileBytes + 2 * kVHalfBytes + kBarBytes;
constexpr uint32_t kOBase = 256;

enum { kEpiPartial = 0, kEpiFinal = 1, kEpiFold = 2, kEpiFoldFinal = 3 };   // as attn_fwd_sm100.cu

template <int kEpi>
__global__ void __launch_bounds__(kThreads, 1)
attn_chunk_fwd_mla_kernel(const __grid_constant__ CUtensorMap map_q, const __grid_constant__ CUtensorMap map_k,
                          const __grid_constant__ CUtensorMap map_v, void* o_out, float* lse_out, const float* o_acc,
                          const float* lse_acc, int Nq, int nk_stride, int k_off, int n_kv, int k_tail,
                          float scale_log2) {
  constexpr bool kFold = kEpi == kEpiFold || kEpi == kEpiFoldFinal;
  constexpr bool kOutBf16 = kEpi == kEpiFinal || kEpi == kEpiFoldFinal;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t* sQ = smem;
  uint8_t* sK = sQ + 2 * kQkTileBytes;
  uint8_t* sV = sK + kKStages * kQkTileBytes;               // [2 halves][2 panels][64 keys][128 B]
  uint64_t* bars = reinterpret_cast<uint64_t*>(sV + 2 * kVHalfBytes);
  uint64_t* q_full = bars;                 // [2]
  uint64_t* s_full = bars + 2;             // [2]  MMA -> softmax: S_t(j) in TMEM
  uint64_t* p_full = bars + 4;             // [2][2] softmax -> MMA: half h of P_t(j) in TMEM
  uint64_t* o_full = bars + 8;             // [2]
  uint64_t* k_full = bars + 10;            // [kKStages]
  uint64_t* k_empty = bars + 12;
  uint64_t* v_full = bars + 14;            // [2] half h of V_j
  uint64_t* v_empty = bars + 16;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 18);

  const int warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0);
  const int lane = threadIdx.x & 31;
  const int bh = blockIdx.y;
  // Any sequence length (as attn_fwd_sm100.cu): q, k, v are [BH][rows][.] tensor maps, so tiles that run past the end of a
  // head read zeros; such query rows are computed and never stored, such keys (k_tail of the last key tile exist) are masked.
  const int q_in = blockIdx.x * (2 * kBlockM);              // first query row of the CTA within its head
  const int q_row0 = bh * Nq + q_in;                        // ... in the flat [BH*Nq] arrays

  if (threadIdx.x == 0) {
    for (int i = 0; i < 2; ++i) {
      mbar_init(&q_full[i], 1);
      mbar_init(&s_full[i], 1);
      mbar_init(&p_full[2 * i], kBlockM);
      mbar_init(&p_full[2 * i + 1], kBlockM);
      mbar_init(&o_full[i], 1);
      mbar_init(&k_full[i], 1);
      mbar_init(&k_empty[i], 1);
      mbar_init(&v_full[i], 1);
      mbar_init(&v_empty[i], 1);
    }
    fence_mbar_init();
  }
  if (warp == 8) {
    if (lane == 0) {
      prefetch_tmap(&map_q);
      prefetch_tmap(&map_k);
      prefetch_tmap(&map_v);
    }
    tmem_alloc<512>(tmem_slot);
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_slot;

  if (warp == 8) {
    setmaxnreg_dec<kAuxRegs>();
    // ------------------------------------------------------------------ TMA producer
    // push order: Q_0 K_0 Q_1 | K_1 V_0.h0 V_0.h1 | K_2 V_1.h0 V_1.h1 | ...  (K_{j+1} ahead of V_j: its slot was freed by
    // S_1(j-1), long before tile 1's P V MMAs of step j-1 free the halves of V)
    const bool leader = elect_one();
    const uint64_t pol_q = policy_evict_first();
    const uint64_t pol_kv = policy_evict_last();
    auto load_qk = [&](uint8_t* dst, const CUtensorMap* map, uint64_t* bar, int row, uint64_t pol) {
      if (leader) {
        mbar_arrive_expect_tx(bar, kQkTileBytes);
#pragma unroll
        for (int p = 0; p < kDqk / 64; ++p) tma_load_3d(dst + p * kPanelBytes, map, bar, p * 64, row, bh, pol);
      }
      __syncwarp();
    };
    auto push_k = [&](int j) {
      const int st = j % kKStages;
      mbar_wait_relaxed(&k_empty[st], ((j / kKStages) & 1) ^ 1);
      load_qk(sK + st * kQkTileBytes, &map_k, &k_full[st], k_off + j * kBlockN, pol_kv);
    };
    load_qk(sQ, &map_q, &q_full[0], q_in, pol_q);
    push_k(0);
    load_qk(sQ + kQkTileBytes, &map_q, &q_full[1], q_in + kBlockM, pol_q);
    for (int j = 0; j < n_kv; ++j) {
      if (j + 1 < n_kv) push_k(j + 1);
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        mbar_wait_relaxed(&v_empty[h], (j & 1) ^ 1);
        if (leader) {
          mbar_arrive_expect_tx(&v_full[h], kVHalfBytes);
#pragma unroll
          for (int p = 0; p < kDv / 64; ++p)       // map_v's box is 64 keys x 64 columns
            tma_load_3d(sV + h * kVHalfBytes + p * kVHalfPanelBytes, &map_v, &v_full[h], p * 64,
                        k_off + j * kBlockN + h * 64, bh, pol_kv);
        }
        __syncwarp();
      }
    }
  } else if (warp == 9) {
    // ------------------------------------------------------------------ MMA issuer
    setmaxnreg_dec<kAuxRegs>();
    const bool leader = elect_one();
    constexpr uint32_t idesc_s = make_idesc_bf16(kBlockM, kBlockN, 0, 0);    // Q (K-major) x K^T (K-major)
    constexpr uint32_t idesc_o = make_idesc_bf16(kBlockM, kDv, 0, 1);        // P (TMEM) x V (MN-major)
    const uint32_t q_addr = smem_u32(sQ), k_addr = smem_u32(sK), v_addr = smem_u32(sV);
    auto commit = [&](uint64_t* bar) {
      if (leader) mma_commit(bar);
      __syncwarp();
    };
    // S_t(j) = Q_t K_j^T: 12 K-steps over three panels
    auto issue_s = [&](int t, int j) {
      const int st = j % kKStages;
      if (t == 0) {
        mbar_wait(&k_full[st], (j / kKStages) & 1);
        tc_fence_after();
      }
      if (j == 0) {
        mbar_wait(&q_full[t], 0);
        tc_fence_after();
      }
      const uint32_t a0 = q_addr + t * kQkTileBytes, b0 = k_addr + st * kQkTileBytes;
      if (leader) {
#pragma unroll
        for (int k = 0; k < kDqk / 16; ++k) {
          const uint32_t off = (k >> 2) * kPanelBytes + (k & 3) * 32;
          mma_ss(tmem + t * kBlockN, make_smem_desc_sw128(a0 + off, 16, 1024), make_smem_desc_sw128(b0 + off, 16, 1024),
                 idesc_s, k > 0);
        }
        mma_commit(&s_full[t]);
      }
      __syncwarp();
      if (t == 1) commit(&k_empty[st]);
    };
    // O_t (+)= P_t(j)[:, 64h .. 64h+64) V_j[64h .. 64h+64, :]: V half h = [2 panels][64 keys][128 B], MN-major B operand
    auto issue_o = [&](int t, int h, bool accumulate) {
      const uint32_t b0 = v_addr + h * kVHalfBytes;
      if (leader) {
#pragma unroll
        for (int kk = 0; kk < 4; ++kk)
          mma_ts(tmem + kOBase + t * kDv, tmem + t * kBlockN + (h * 4 + kk) * 8,
                 make_smem_desc_sw128(b0 + kk * 2048, kVHalfPanelBytes, 1024), idesc_o, accumulate || kk > 0);
      }
      __syncwarp();
    };
    issue_s(0, 0);
    issue_s(1, 0);
    for (int j = 0; j < n_kv; ++j) {
#pragma unroll
      for (int t = 0; t < 2; ++t) {
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          if (t == 0) {
            mbar_wait(&v_full[h], j & 1);
            tc_fence_after();
          }
          mbar_wait(&p_full[2 * t + h], j & 1);
          tc_fence_after();
          issue_o(t, h, j > 0 || h > 0);
          if (t == 1) commit(&v_empty[h]);                   // both query tiles are done with this half of V_j
        }
        if (j + 1 == n_kv) commit(&o_full[t]);
        if (j + 1 < n_kv) issue_s(t, j + 1);
      }
    }
  } else if (warp < 8) {
    // ------------------------------------------------------------------ softmax warpgroups (as the d = 128 kernel)
    setmaxnreg_inc<kSoftmaxRegs>();
    const int t = warp >> 2;
    const int row_t = (warp & 3) * 32 + lane;
    const uint32_t lane_off = static_cast<uint32_t>((warp & 3) * 32) << 16;
    const uint32_t tS = tmem + t * kBlockN + lane_off;
    const uint32_t tO = tmem + kOBase + t * kDv + lane_off;
    const float2 sc2 = make_float2(scale_log2, scale_log2);
    const size_t row = static_cast<size_t>(q_row0) + t * kBlockM + row_t;
    const bool row_valid = q_in + t * kBlockM + row_t < Nq;
    float lse_prev = 0.f;
    if (kFold && row_valid) lse_prev = lse_acc[row];
    float m_raw = -CUDART_INF_F, m_sc = -CUDART_INF_F, l = 0.f;
    for (int j = 0; j < n_kv; ++j) {
      mbar_wait(&s_full[t], j & 1);
      tc_fence_after();
      uint32_t s[kBlockN];
      auto piece = [&](int c) -> uint32_t(&)[32] { return *reinterpret_cast<uint32_t(*)[32]>(&s[c * 32]); };
      auto piece_max = [&](int c, float& a, float& b) {
#pragma unroll
        for (int i = 0; i < 32; i += 4) {
          a = fmax3(a, __uint_as_float(s[c * 32 + i]), __uint_as_float(s[c * 32 + i + 1]));
          b = fmax3(b, __uint_as_float(s[c * 32 + i + 2]), __uint_as_float(s[c * 32 + i + 3]));
        }
      };
      float mx0 = -CUDART_INF_F, mx1 = -CUDART_INF_F, mx2 = -CUDART_INF_F, mx3 = -CUDART_INF_F;
      tmem_ld_x32(tS, piece(0));
      tmem_wait_ld_x32(piece(0));
      tmem_ld_x32(tS + 32, piece(1));
      piece_max(0, mx0, mx1);
      tmem_wait_ld_x32(piece(1));
      tmem_ld_x32(tS + 64, piece(2));
      piece_max(1, mx2, mx3);
      tmem_wait_ld_x32(piece(2));
      tmem_ld_x32(tS + 96, piece(3));
      piece_max(2, mx0, mx1);
      tmem_wait_ld_x32(piece(3));
      piece_max(3, mx2, mx3);
      if (k_tail != 0 && j == n_kv - 1) {                    // warp-uniform: the last key tile of a ragged head
#pragma unroll
        for (int c = 0; c < kBlockN; ++c)
          if (c >= k_tail) s[c] = 0xff800000u;               // -inf
        mx0 = mx1 = mx2 = mx3 = -CUDART_INF_F;
        piece_max(0, mx0, mx1);
        piece_max(1, mx2, mx3);
        piece_max(2, mx0, mx1);
        piece_max(3, mx2, mx3);
      }
      const float mx = fmaxf(fmaxf(mx0, mx1), fmaxf(mx2, mx3));
      const bool grow = (mx - m_raw) * scale_log2 > kRescaleThreshold;
      if (__any_sync(0xffffffffu, grow)) {
        const float m_new = fmaxf(m_raw, mx);
        const float alpha = ex2((m_raw - m_new) * scale_log2);   // 0 on the first tile (m_raw = -inf)
        l *= alpha;
        if (j > 0) {        // (s_full(j) was committed behind O_t += P_t(j-1) V: O_t is complete and may be rescaled in place)
#pragma unroll
          for (int c = 0; c < kDv / 32; ++c) {
            uint32_t o[32];
            tmem_ld_x32(tO + c * 32, o);
            tmem_wait_ld_x32(o);
#pragma unroll
            for (int i = 0; i < 32; ++i) o[i] = __float_as_uint(__uint_as_float(o[i]) * alpha);
            tmem_st_x32(tO + c * 32, o);
          }
        }
        m_raw = m_new;
        m_sc = m_new * scale_log2;
      }
      const float2 nm2 = make_float2(-m_sc, -m_sc);
      float2 la = make_float2(0.f, 0.f), lb = make_float2(0.f, 0.f);
#pragma unroll
      for (int c = 0; c < kBlockN / 32; ++c) {
        uint32_t pk[16];
#pragma unroll
        for (int i = 0; i < 32; i += 4) {
          const float2 x0 = ffma2(make_float2(__uint_as_float(s[c * 32 + i]), __uint_as_float(s[c * 32 + i + 1])), sc2, nm2);
          const float2 x1 = ffma2(make_float2(__uint_as_float(s[c * 32 + i + 2]), __uint_as_float(s[c * 32 + i + 3])), sc2, nm2);
          const float2 p0 = make_float2(ex2(x0.x), ex2(x0.y));
          const float2 p1 = make_float2(ex2(x1.x), ex2(x1.y));
          la = fadd2(la, p0);
          lb = fadd2(lb, p1);
          pk[i / 2] = pack_bf16x2(p0.x, p0.y);
          pk[i / 2 + 1] = pack_bf16x2(p1.x, p1.y);
        }
        tmem_st_x16(tS + c * 16, pk);
        if (c & 1) {                       // 64 keys of P are in TMEM: let the tensor core start on them
          tmem_wait_st();
          tc_fence_before();
          mbar_arrive(&p_full[2 * t + (c >> 1)]);
        }
      }
      l += (la.x + la.y) + (lb.x + lb.y);
    }
    // ---- chunk epilogue: loc_out = O / l, loc_lse = m*scale + ln l; Eq. 5 fold with the running (o_acc, lse_acc)
    mbar_wait(&o_full[t], 0);
    tc_fence_after();
    float lse_row = (m_sc + lg2(l)) * 0.6931471805599453f;
    float cb = 1.0f / l, ca = 0.f;
    if (kFold) {
      const float m = fmaxf(lse_prev, lse_row);
      const float wa = ex2((lse_prev - m) * 1.4426950408889634f), wb = ex2((lse_row - m) * 1.4426950408889634f);
      const float den = wa + wb, r = 1.0f / den;
      ca = wa * r;
      cb *= wb * r;
      lse_row = m + lg2(den) * 0.6931471805599453f;
    }
#pragma unroll
    for (int c = 0; c < kDv / 32; ++c) {
      uint32_t o[32];
      tmem_ld_x32(tO + c * 32, o);
      float4 acc[8];
      if (kFold) {
        const float4* src = reinterpret_cast<const float4*>(o_acc + row * kDv + c * 32);
#pragma unroll
        for (int i = 0; i < 8; ++i) acc[i] = row_valid ? __ldcs(src + i) : make_float4(0.f, 0.f, 0.f, 0.f);
      }
      tmem_wait_ld();
      float r[32];
#pragma unroll
      for (int i = 0; i < 32; ++i) r[i] = __uint_as_float(o[i]) * cb;
      if (kFold) {
#pragma unroll
        for (int i = 0; i < 8; ++i) {
          r[i * 4 + 0] = fmaf(ca, acc[i].x, r[i * 4 + 0]);
          r[i * 4 + 1] = fmaf(ca, acc[i].y, r[i * 4 + 1]);
          r[i * 4 + 2] = fmaf(ca, acc[i].z, r[i * 4 + 2]);
          r[i * 4 + 3] = fmaf(ca, acc[i].w, r[i * 4 + 3]);
        }
      }
      if (!row_valid) continue;
      if (kOutBf16) {
        uint4* dst = reinterpret_cast<uint4*>(static_cast<__nv_bfloat16*>(o_out) + row * kDv + c * 32);
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          uint4 u;
          u.x = pack_bf16x2(r[i * 8 + 0], r[i * 8 + 1]);
          u.y = pack_bf16x2(r[i * 8 + 2], r[i * 8 + 3]);
          u.z = pack_bf16x2(r[i * 8 + 4], r[i * 8 + 5]);
          u.w = pack_bf16x2(r[i * 8 + 6], r[i * 8 + 7]);
          dst[i] = u;
        }
      } else {
        float4* dst = reinterpret_cast<float4*>(static_cast<float*>(o_out) + row * kDv + c * 32);
#pragma unroll
        for (int i = 0; i < 8; ++i) dst[i] = make_float4(r[i * 4], r[i * 4 + 1], r[i * 4 + 2], r[i * 4 + 3]);
      }
    }
    if (row_valid) lse_out[row] = lse_row;
  } else {
    setmaxnreg_dec<kAuxRegs>();
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 8) tmem_dealloc<512>(tmem);
}

template <int kEpi>
cudaError_t launch_t(const CUtensorMap& mq, const CUtensorMap& mk, const CUtensorMap& mv, void* o_out, float* lse_out,
                     const float* o_acc, const float* lse_acc, int BH, int Nq, int nk_stride, int k_off, int nk,
                     float scale, cudaStream_t stream) {
  auto kern = attn_chunk_fwd_mla_kernel<kEpi>;
  static unsigned char configured[kMaxDevices];
  if (cudaError_t e = set_max_dyn_smem_once(kern, kSmemBytes, configured); e != cudaSuccess) return e;
  dim3 grid((Nq + 2 * kBlockM - 1) / (2 * kBlockM), BH);
  kern<<<grid, kThreads, kSmemBytes, stream>>>(mq, mk, mv, o_out, lse_out, o_acc, lse_acc, Nq, nk_stride, k_off,
                                               (nk + kBlockN - 1) / kBlockN, nk % kBlockN, scale * 1.4426950408889634f);
  count_launch();
  return cudaGetLastError();
}

}  // namespace

cudaError_t launch_attn_chunk_fwd_mla_sm100(const void* q, const void* k, const void* v, void* o_out, float* lse_out,
                                            const float* o_acc, const float* lse_acc, int BH, int Nq, int nk_stride,
                                            int k_off, int nk, float scale, int epilogue, cudaStream_t stream) {
  CUtensorMap mq, mk, mv;
  const CUtensorMapDataType dt = CU_TENSOR_MAP_DATA_TYPE_BFLOAT16;
  if (nk % kBlockN && k_off + nk != nk_stride) return cudaErrorInvalidValue;   // only the head's last key tile may be ragged
  if (!make_tmap_3d(&mq, q, dt, 2, BH, Nq, kDqk, 128, 64, kSwizzle128B) ||
      !make_tmap_3d(&mk, k, dt, 2, BH, nk_stride, kDqk, 128, 64, kSwizzle128B) ||
      !make_tmap_3d(&mv, v, dt, 2, BH, nk_stride, kDv, 64, 64, kSwizzle128B))      // half tiles: 64 keys
    return cudaErrorInvalidValue;
  switch (epilogue) {
    case kFwdEpiPartial:
      return launch_t<kEpiPartial>(mq, mk, mv, o_out, lse_out, o_acc, lse_acc, BH, Nq, nk_stride, k_off, nk, scale, stream);
    case kFwdEpiFinal:
      return launch_t<kEpiFinal>(mq, mk, mv, o_out, lse_out, o_acc, lse_acc, BH, Nq, nk_stride, k_off, nk, scale, stream);
    case kFwdEpiFold:
      return launch_t<kEpiFold>(mq, mk, mv, o_out, lse_out, o_acc, lse_acc, BH, Nq, nk_stride, k_off, nk, scale, stream);
    default:
      return launch_t<kEpiFoldFinal>(mq, mk, mv, o_out, lse_out, o_acc, lse_acc, BH, Nq, nk_stride, k_off, nk, scale, stream);
  }
}

}  // namespace ringx
