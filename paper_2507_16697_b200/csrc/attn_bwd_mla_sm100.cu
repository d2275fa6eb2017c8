// attn_bwd_mla_sm100.cu -- one KV-chunk pass of the backward for multi-head LATENT attention shapes (SURVEY.md §8(f)
// NEXT-3): d_qk = 192 (128 "nope" + 64 rotary dimensions), d_v = 128.  Same mathematics as
// attn_bwd_sm100.cu (the derivative of Eq. 1 with P recomputed from the saved global LSE, reading g8; data flow of
// PAPER.md:143), with a score contraction that is longer than the value width:
//   S^T  = K_j Q_s^T   (192)        P^T  = exp2(scale*log2e * S^T - lse2_s)
//   dP^T = V_j dO_s^T  (128)        dS^T = P^T o (scale*dP^T - scale*D_s)
//   dV_j += P^T dO_s   [128 x 128]  dK_j += dS^T Q_s  [128 x 192]     dQ_s += dS K_j  [64 x 192]
//
// What d_qk = 192 changes.  A CTA still owns one 128-key tile and keeps dK_j, dV_j in TMEM for its whole walk over the
// queries (written once, atomic-free) -- but those are 192 + 128 = 320 of the 512 TMEM columns, and K_j, V_j are 80 KB
// of shared memory, so neither two 128-column score tiles nor two 48 KB Q tiles fit next to them.  The walk therefore
// advances in SUB-TILES of 64 queries: S^T, dP^T are [128 keys x 64 queries] (64 columns each), a Q sub-tile is 24 KB.
// dQ is computed TRANSPOSED, dQ_s^T = K_j^T dS^T ([d x 64]: M = the feature index, which can be 128; M = 64 queries
// would halve the tensor rate), in two M = 128 pieces -- features [0,128) and [64,192), the second one's lanes 64..127
// being features [128,192) (its lanes 0..63 repeat features [64,128) and are dropped) -- and reduce-added by TMA into a
// TRANSPOSED fp32 accumulator dq_acc^T [BH, 192, Nq]; `dq_transpose_convert_kernel` turns it into dq [BH, Nq, 192] bf16.
//
// TMEM columns: S^T [0,64) (P^T, bf16, over columns [0,16) and [32,48)), dP^T [64,128) (dQ^T piece B overlays it and
// is drained before the next dP^T is issued), dQ^T piece A [128,192), dV [192,320), dK [320,512).
// Roles (512 threads, as attn_bwd_sm100.cu): warps 0-7 compute (thread = key row = TMEM lane; warps 0-3 take query
// columns 0-31 of the sub-tile, warps 4-7 columns 32-63), warps 8-11 dQ^T drain (thread = feature row), warp 12 TMA
// producer, warp 13 MMA issuer, warps 14-15 idle.  Pipeline as there: the tensor core runs {dV(s), S^T(s+1)} behind
// phase A and {dQ^T(s), dK(s), dP^T(s+1)} behind phase B.
#include "kernels.cuh"

namespace ringx {
namespace {

using namespace ptx;

constexpr int kKeys = 128;                       // keys per CTA = TMEM lanes
constexpr int kSub = 64;                         // queries per step
constexpr int kDqk = 192, kDv = 128;
constexpr int kThreads = 512;
constexpr int kComputeRegs = 176, kDrainRegs = 96, kAuxRegs = 40;
constexpr int kKPanel = 128 * 128;               // [128 rows][64 bf16], 128B-swizzled
constexpr int kQPanel = 64 * 128;                // [64 rows][64 bf16]
constexpr int kKBytes = (kDqk / 64) * kKPanel;   // K_j: 48 KB
constexpr int kVBytes = (kDv / 64) * kKPanel;    // V_j: 32 KB
constexpr int kQBytes = (kDqk / 64) * kQPanel;   // Q_s: 24 KB
constexpr int kDoBytes = (kDv / 64) * kQPanel;   // dO_s: 16 KB
constexpr int kQStageBytes = kQBytes + 1024;     // Q_s | lse2[64] | D[64]
constexpr int kQStages = 2, kDoStages = 2;
constexpr int kDsBytes = kKPanel;                // dS^T [128 keys][64 queries] bf16
constexpr int kDqPanelBytes = 128 * 128;         // staging: [128 feature rows][32 fp32 queries], 128B-swizzled
constexpr int kSmemBytes = 1024 + kKBytes + kVBytes + kQStages * kQStageBytes + kDoStages * kDoBytes + kDsBytes +
                           2 * kDqPanelBytes + 256;
constexpr uint32_t tS = 0, tDP = 64, tDQ = 128, tDV = 192, tDK = 320;

__global__ void __launch_bounds__(kThreads, 1)
attn_chunk_bwd_mla_kernel(const __grid_constant__ CUtensorMap map_q, const __grid_constant__ CUtensorMap map_k,
                          const __grid_constant__ CUtensorMap map_v, const __grid_constant__ CUtensorMap map_do,
                          const __grid_constant__ CUtensorMap map_dq_a, const __grid_constant__ CUtensorMap map_dq_b,
                          const float* __restrict__ lse2, const float* __restrict__ Dvec, void* __restrict__ dk,
                          void* __restrict__ dv, int dkv_f32, int N, int n_stat, int nk_stride, int k_off,
                          float scale_log2, float scale, const float* __restrict__ dq_qs) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t* sK = smem;
  uint8_t* sV = sK + kKBytes;
  uint8_t* sQ = sV + kVBytes;                          // [kQStages] Q_s | lse2_s | D_s
  uint8_t* sDo = sQ + kQStages * kQStageBytes;         // [kDoStages] dO_s
  uint8_t* sDs = sDo + kDoStages * kDoBytes;
  uint8_t* sDq = sDs + kDsBytes;                       // 2 staging panels for the dQ^T reduce-add
  uint64_t* bars = reinterpret_cast<uint64_t*>(sDq + 2 * kDqPanelBytes);
  uint64_t* kv_full = bars;          // TMA -> MMA: K_j, V_j
  uint64_t* s_full = bars + 1;       // MMA -> compute: S^T(s)
  uint64_t* dp_full = bars + 2;      // MMA -> compute: dP^T(s)
  uint64_t* p_full = bars + 3;       // compute -> MMA: P^T(s) in TMEM, S^T(s) consumed            (8 arrivals: one per warp)
  uint64_t* ds_full = bars + 4;      // compute -> MMA: dS^T(s) in smem, dP^T(s) consumed          (8 arrivals)
  uint64_t* ds_empty = bars + 5;     // MMA -> compute: dK(s), dQ^T(s) have read dS^T(s)
  uint64_t* dq_full = bars + 6;      // MMA -> drain: both pieces of dQ^T(s) in TMEM
  uint64_t* dq_empty = bars + 7;     // drain -> MMA: dQ^T(s) in registers                          (4 arrivals)
  uint64_t* dkv_full = bars + 8;     // MMA -> compute: dK_j, dV_j complete
  uint64_t* q_full = bars + 9;       // [kQStages]
  uint64_t* q_empty = q_full + kQStages;
  uint64_t* do_full = q_empty + kQStages;     // [kDoStages]
  uint64_t* do_empty = do_full + kDoStages;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(do_empty + kDoStages);

  const int warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0);
  const int lane = threadIdx.x & 31;
  const int bh = blockIdx.y;
  // Any sequence length (as attn_bwd_sm100.cu): q, dO, k, v are [BH][rows][.] tensor maps (rows past the end of a head read
  // as zeros), lse2 / D are [BH][n_stat] with lse2 = +inf in the padding (P = 0 for query rows that do not exist), keys past
  // the end get P = 0 by a select and their dK, dV rows are not stored, the dQ^T reduce-add skips the missing queries.
  const int n_s = (N + kSub - 1) / kSub;
  const int q_row0 = bh * N;                                        // rows of this head in the flat [BH*N] array dq_qs
  const int s_row0 = bh * n_stat;                                   // ... in lse2, D
  const int k_in = k_off + blockIdx.x * kKeys;                      // first key row of my tile within the head
  const int k_row0 = bh * nk_stride + k_in;                         // ... in the flat [BH*nk_stride, .] arrays dK, dV

  if (threadIdx.x == 0) {
    mbar_init(kv_full, 1);
    mbar_init(s_full, 1);
    mbar_init(dp_full, 1);
    mbar_init(p_full, 8);
    mbar_init(ds_full, 8);
    mbar_init(ds_empty, 1);
    mbar_init(dq_full, 1);
    mbar_init(dq_empty, 4);
    mbar_init(dkv_full, 1);
    for (int i = 0; i < kQStages; ++i) {
      mbar_init(&q_full[i], 1);
      mbar_init(&q_empty[i], 1);
    }
    for (int i = 0; i < kDoStages; ++i) {
      mbar_init(&do_full[i], 1);
      mbar_init(&do_empty[i], 1);
    }
    fence_mbar_init();
  }
  if (warp == 12) {
    if (lane == 0) {
      prefetch_tmap(&map_q);
      prefetch_tmap(&map_k);
      prefetch_tmap(&map_v);
      prefetch_tmap(&map_do);
      prefetch_tmap(&map_dq_a);
      prefetch_tmap(&map_dq_b);
    }
    tmem_alloc<512>(tmem_slot);
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_slot;

  if (warp == 12) {
    // ------------------------------------------------------------------ TMA producer
    setmaxnreg_dec<kAuxRegs>();
    const bool leader = elect_one();
    const uint64_t pol_kv = policy_evict_first();
    const uint64_t pol_q = policy_evict_last();      // Q/dO sub-tiles are re-read by every CTA of the head
    if (leader) {
      mbar_arrive_expect_tx(kv_full, kKBytes + kVBytes);
#pragma unroll
      for (int p = 0; p < kDqk / 64; ++p) tma_load_3d(sK + p * kKPanel, &map_k, kv_full, p * 64, k_in, bh, pol_kv);
#pragma unroll
      for (int p = 0; p < kDv / 64; ++p) tma_load_3d(sV + p * kKPanel, &map_v, kv_full, p * 64, k_in, bh, pol_kv);
    }
    __syncwarp();
    auto load_q = [&](int s, int st) {
      if (leader) {
        uint8_t* dst = sQ + st * kQStageBytes;
        mbar_arrive_expect_tx(&q_full[st], kQBytes + 512);
#pragma unroll
        for (int p = 0; p < kDqk / 64; ++p) tma_load_3d(dst + p * kQPanel, &map_q, &q_full[st], p * 64, s * kSub, bh, pol_q);
        bulk_load_1d(dst + kQBytes, lse2 + s_row0 + s * kSub, 256, &q_full[st]);
        bulk_load_1d(dst + kQBytes + 256, Dvec + s_row0 + s * kSub, 256, &q_full[st]);
      }
      __syncwarp();
    };
    load_q(0, 0);
    int qs = 1, qph = 0, ds = 0, dph = 0;
    for (int s = 0; s < n_s; ++s) {
      // dO_s: its slot is free once dV(s - kDoStages) has read it
      mbar_wait_relaxed(&do_empty[ds], dph ^ 1);
      if (leader) {
        mbar_arrive_expect_tx(&do_full[ds], kDoBytes);
#pragma unroll
        for (int p = 0; p < kDv / 64; ++p)
          tma_load_3d(sDo + ds * kDoBytes + p * kQPanel, &map_do, &do_full[ds], p * 64, s * kSub, bh, pol_q);
      }
      __syncwarp();
      if (++ds == kDoStages) { ds = 0; dph ^= 1; }
      // Q_{s+1}: its slot is free once dK(s + 1 - kQStages) has read it
      if (s + 1 < n_s) {
        mbar_wait_relaxed(&q_empty[qs], qph ^ 1);
        load_q(s + 1, qs);
        if (++qs == kQStages) { qs = 0; qph ^= 1; }
      }
    }
  } else if (warp == 13) {
    // ------------------------------------------------------------------ MMA issuer
    setmaxnreg_dec<kAuxRegs>();
    const bool leader = elect_one();
    constexpr uint32_t idesc_st = make_idesc_bf16(kKeys, kSub, 0, 0);    // K_j / V_j (K-major) x Q_s^T / dO_s^T (K-major)
    constexpr uint32_t idesc_dv = make_idesc_bf16(kKeys, kDv, 0, 1);     // P^T (TMEM) x dO_s (MN-major)
    constexpr uint32_t idesc_dk = make_idesc_bf16(kKeys, kDqk, 0, 1);    // dS^T (K-major) x Q_s (MN-major)
    constexpr uint32_t idesc_dq = make_idesc_bf16(128, kSub, 1, 1);      // K_j^T (MN-major) x dS^T (MN-major)
    const uint32_t k_addr = smem_u32(sK), v_addr = smem_u32(sV), ds_addr = smem_u32(sDs);
    const uint32_t q_base = smem_u32(sQ), do_base = smem_u32(sDo);
    auto kmajor128 = [](uint32_t base, int k) {   // K-step k of a K-major tile of 128-row panels
      return make_smem_desc_sw128(base + (k >> 2) * kKPanel + (k & 3) * 32, 16, 1024);
    };
    auto kmajor64 = [](uint32_t base, int k) {    // ... of 64-row panels
      return make_smem_desc_sw128(base + (k >> 2) * kQPanel + (k & 3) * 32, 16, 1024);
    };
    auto mnmajor = [](uint32_t base, int k, uint32_t panel) {   // K-step k (16 rows) of a [K rows][MN contiguous] tile
      return make_smem_desc_sw128(base + k * 2048, panel, 1024);
    };
    auto commit = [&](uint64_t* bar) {
      if (leader) mma_commit(bar);
      __syncwarp();
    };
    auto issue_st = [&](uint32_t q_addr) {
      if (leader) {
#pragma unroll
        for (int k = 0; k < kDqk / 16; ++k)
          mma_ss(tmem + tS, kmajor128(k_addr, k), kmajor64(q_addr, k), idesc_st, k > 0);
        mma_commit(s_full);
      }
      __syncwarp();
    };
    auto issue_dpt = [&](uint32_t do_addr) {
      if (leader) {
#pragma unroll
        for (int k = 0; k < kDv / 16; ++k)
          mma_ss(tmem + tDP, kmajor128(v_addr, k), kmajor64(do_addr, k), idesc_st, k > 0);
        mma_commit(dp_full);
      }
      __syncwarp();
    };
    mbar_wait(kv_full, 0);
    mbar_wait(&q_full[0], 0);
    tc_fence_after();
    issue_st(q_base);
    mbar_wait(&do_full[0], 0);
    tc_fence_after();
    issue_dpt(do_base);
    int qs = 0, qph = 0, ds = 0, dph = 0;
    for (int s = 0; s < n_s; ++s) {
      const uint32_t q_addr = q_base + qs * kQStageBytes, do_addr = do_base + ds * kDoBytes;
      const int cur_qs = qs, cur_ds = ds;
      if (++qs == kQStages) { qs = 0; qph ^= 1; }
      if (++ds == kDoStages) { ds = 0; dph ^= 1; }
      const bool more = s + 1 < n_s;
      // ---- behind phase A: dV += P^T(s) dO_s, then S^T(s+1)
      mbar_wait(p_full, s & 1);
      tc_fence_after();
      if (leader) {
#pragma unroll
        for (int k = 0; k < kSub / 16; ++k)
          mma_ts(tmem + tDV, tmem + tS + (k >> 1) * 32 + (k & 1) * 8, mnmajor(do_addr, k, kQPanel), idesc_dv,
                 s > 0 || k > 0);
        mma_commit(&do_empty[cur_ds]);
      }
      __syncwarp();
      if (more) {
        mbar_wait(&q_full[qs], qph);
        tc_fence_after();
        issue_st(q_base + qs * kQStageBytes);
      }
      // ---- behind phase B: dQ^T(s) = K_j^T dS^T(s) in two pieces, dK += dS^T(s) Q_s, then dP^T(s+1)
      mbar_wait(ds_full, s & 1);
      tc_fence_after();
      if (leader) {
#pragma unroll
        for (int k = 0; k < kKeys / 16; ++k)       // piece A: features [0,128)
          mma_ss(tmem + tDQ, mnmajor(k_addr, k, kKPanel), mnmajor(ds_addr, k, kKPanel), idesc_dq, k > 0);
#pragma unroll
        for (int k = 0; k < kKeys / 16; ++k)       // piece B: features [64,192) over the (consumed) dP^T columns
          mma_ss(tmem + tDP, mnmajor(k_addr + kKPanel, k, kKPanel), mnmajor(ds_addr, k, kKPanel), idesc_dq, k > 0);
        mma_commit(dq_full);
#pragma unroll
        for (int k = 0; k < kSub / 16; ++k)
          mma_ss(tmem + tDK, kmajor128(ds_addr, k), mnmajor(q_addr, k, kQPanel), idesc_dk, s > 0 || k > 0);
        mma_commit(ds_empty);
        mma_commit(&q_empty[cur_qs]);
      }
      __syncwarp();
      if (more) {
        mbar_wait(&do_full[ds], dph);
        mbar_wait(dq_empty, s & 1);               // dQ^T(s) piece B sits in the dP^T columns until drained
        tc_fence_after();
        issue_dpt(do_base + ds * kDoBytes);
      }
    }
    commit(dkv_full);
  } else if (warp < 8) {
    // ------------------------------------------------------------------ compute warps
    setmaxnreg_inc<kComputeRegs>();
    const int half = warp >> 2;                                  // which 32 query columns of the sub-tile
    const int row = (warp & 3) * 32 + lane;                      // key row of the tile = TMEM lane
    const uint32_t lane_off = static_cast<uint32_t>((warp & 3) * 32) << 16;
    const uint32_t tSm = tmem + tS + lane_off + half * 32;       // my S^T columns; P^T goes to the first 16 of them
    const uint32_t tDPm = tmem + tDP + lane_off + half * 32;
    uint8_t* ds_row = sDs + row * 128;
    const float2 sc2 = make_float2(scale_log2, scale_log2);
    const float2 scl2 = make_float2(scale, scale);               // dS^T carries `scale` (Dvec holds scale * D_i)
    const bool key_valid = k_in + row < nk_stride;
    int stage = 0, phase = 0;
    for (int s = 0; s < n_s; ++s) {
      const float4* stats = reinterpret_cast<const float4*>(sQ + stage * kQStageBytes + kQBytes);
      const float4* lse4 = stats + half * 8;                     // lse2 of my 32 query columns
      const float4* d4 = stats + 16 + half * 8;                  // D of my 32 query columns
      mbar_wait(&q_full[stage], phase);
      if (++stage == kQStages) { stage = 0; phase ^= 1; }
      // ---- phase A: P^T = exp2(scale_log2 * S^T - lse2)
      float4 aux[8];
#pragma unroll
      for (int g = 0; g < 8; ++g) aux[g] = ld_shared_v4(lse4 + g);
      mbar_wait(s_full, s & 1);
      tc_fence_after();
      float2 p[16];
      {
        uint32_t sv[32], pk[16];
        tmem_ld_x32(tSm, sv);
        tmem_wait_ld_x32(sv);
#pragma unroll
        for (int g = 0; g < 8; ++g) {
          const float2 x0 = ffma2(make_float2(__uint_as_float(sv[g * 4 + 0]), __uint_as_float(sv[g * 4 + 1])), sc2,
                                  make_float2(-aux[g].x, -aux[g].y));
          const float2 x1 = ffma2(make_float2(__uint_as_float(sv[g * 4 + 2]), __uint_as_float(sv[g * 4 + 3])), sc2,
                                  make_float2(-aux[g].z, -aux[g].w));
          p[g * 2] = key_valid ? make_float2(ex2(x0.x), ex2(x0.y)) : make_float2(0.f, 0.f);     // (a key past the end of the head)
          p[g * 2 + 1] = key_valid ? make_float2(ex2(x1.x), ex2(x1.y)) : make_float2(0.f, 0.f);
          pk[g * 2] = pack_bf16x2(p[g * 2].x, p[g * 2].y);
          pk[g * 2 + 1] = pack_bf16x2(p[g * 2 + 1].x, p[g * 2 + 1].y);
        }
#pragma unroll
        for (int g = 0; g < 8; ++g) aux[g] = ld_shared_v4(d4 + g);       // phase B's D
        tmem_st_x16(tSm, pk);              // overlays only S^T columns this thread has already loaded
      }
      tmem_wait_st();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(p_full);          // one arrival per warp (8), as in attn_bwd_sm100.cu: 256 separate arrivals are 256 shared-memory atomics
      // ---- phase B: dS^T = P^T o (scale dP^T - scale D), bf16, to shared memory [keys][queries] (128B-swizzled rows)
      mbar_wait(dp_full, s & 1);
      if (s > 0) mbar_wait(ds_empty, (s - 1) & 1);
      tc_fence_after();
      {
        uint32_t dp[32];
        tmem_ld_x32(tDPm, dp);
        tmem_wait_ld_x32(dp);
        float2 t[16];
#pragma unroll
        for (int g = 0; g < 8; ++g) {
          t[g * 2] = ffma2(make_float2(__uint_as_float(dp[g * 4 + 0]), __uint_as_float(dp[g * 4 + 1])), scl2,
                           make_float2(-aux[g].x, -aux[g].y));
          t[g * 2 + 1] = ffma2(make_float2(__uint_as_float(dp[g * 4 + 2]), __uint_as_float(dp[g * 4 + 3])), scl2,
                               make_float2(-aux[g].z, -aux[g].w));
        }
#pragma unroll
        for (int g = 0; g < 4; ++g) {       // 8 queries = one 16-byte chunk of the row
          const int e = g * 4;
          const float2 w0 = fmul2(p[e + 0], t[e + 0]), w1 = fmul2(p[e + 1], t[e + 1]);
          const float2 w2 = fmul2(p[e + 2], t[e + 2]), w3 = fmul2(p[e + 3], t[e + 3]);
          const int chunk = half * 4 + g;
          st_shared_v4(ds_row + ((chunk ^ (row & 7)) << 4), pack_bf16x2(w0.x, w0.y), pack_bf16x2(w1.x, w1.y),
                       pack_bf16x2(w2.x, w2.y), pack_bf16x2(w3.x, w3.y));
        }
      }
      fence_proxy_async_smem();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(ds_full);
    }
    // ---- epilogue: dV_j (warps 0-3, 128 columns) and dK_j (warps 4-7, 192 columns), bf16, written once
    mbar_wait(dkv_full, 0);
    tc_fence_after();
    const int width = half == 0 ? kDv : kDqk;
    const uint32_t tSrc = tmem + (half == 0 ? tDV : tDK) + lane_off;
    const size_t out_off = (static_cast<size_t>(k_row0) + row) * width;
    // bf16 (the single-device result), or fp32 (one device's share of a cross-device sum: RingX_a/b reduce the shares
    // in fp32 and round once)
    for (int c = 0; c < width / 32; ++c) {
      uint32_t r[32];
      tmem_ld_x32(tSrc + c * 32, r);
      tmem_wait_ld();
      if (!key_valid) continue;              // (after the warp-wide TMEM load)
      if (dkv_f32) {
        float4* dst = reinterpret_cast<float4*>(static_cast<float*>(half == 0 ? dv : dk) + out_off + c * 32);
#pragma unroll
        for (int g = 0; g < 8; ++g)
          dst[g] = make_float4(__uint_as_float(r[g * 4]), __uint_as_float(r[g * 4 + 1]), __uint_as_float(r[g * 4 + 2]),
                               __uint_as_float(r[g * 4 + 3]));
      } else {
        uint4* dst = reinterpret_cast<uint4*>(static_cast<__nv_bfloat16*>(half == 0 ? dv : dk) + out_off + c * 32);
#pragma unroll
        for (int g = 0; g < 4; ++g) {
          uint4 u;
          u.x = pack_bf16x2(__uint_as_float(r[g * 8 + 0]), __uint_as_float(r[g * 8 + 1]));
          u.y = pack_bf16x2(__uint_as_float(r[g * 8 + 2]), __uint_as_float(r[g * 8 + 3]));
          u.z = pack_bf16x2(__uint_as_float(r[g * 8 + 4]), __uint_as_float(r[g * 8 + 5]));
          u.w = pack_bf16x2(__uint_as_float(r[g * 8 + 6]), __uint_as_float(r[g * 8 + 7]));
          dst[g] = u;
        }
      }
    }
  } else if (warp < 12) {
    // ------------------------------------------------------------------ dQ^T drain warps (8-11)
    // thread = feature row of a piece = TMEM lane; 64 query columns per piece -> two staging panels [128 rows][32 fp32]
    // -> TMA reduce-add into dq_acc^T [BH*192, Nq].  Piece A = features [0,128): all 128 rows; piece B = features
    // [64,192): only rows 64..127 (features [128,192)) are stored and reduced (box of 64 rows).
    setmaxnreg_dec<kDrainRegs>();
    const int row = (warp & 3) * 32 + lane;
    const uint32_t lane_off = static_cast<uint32_t>((warp & 3) * 32) << 16;
    const bool leader = warp == 8 && elect_one();
    int buf = 0;
    for (int s = 0; s < n_s; ++s) {
      mbar_wait(dq_full, s & 1);
      tc_fence_after();
#pragma unroll
      for (int piece = 0; piece < 2; ++piece) {
        uint32_t r[2][32];
#pragma unroll
        for (int c = 0; c < 2; ++c) tmem_ld_x32(tmem + (piece == 0 ? tDQ : tDP) + lane_off + c * 32, r[c]);
#pragma unroll
        for (int c = 0; c < 2; ++c) tmem_wait_ld_x32(r[c]);
        if (piece == 1) {
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(dq_empty);   // both pieces of dQ^T(s) have left TMEM: hand the columns back
        }
        if (dq_qs) {
          // deterministic mode (attn_bwd_sm100.cu): int32 fixed point; here a thread is a feature row and its 64
          // registers are the 64 queries of the sub-tile, each with its own scale (warp-uniform 16-byte loads)
          const float* qs1 = dq_qs + q_row0 + s * kSub;       // (scalar loads: a ragged head is not 16-byte aligned)
#pragma unroll
          for (int c = 0; c < 2; ++c)
#pragma unroll
            for (int e = 0; e < 32; ++e) {
              const float f = s * kSub + c * 32 + e < N ? __ldg(qs1 + c * 32 + e) : 0.f;
              r[c][e] = static_cast<uint32_t>(__float2int_rn(__uint_as_float(r[c][e]) * f));
            }
        }
#pragma unroll
        for (int c = 0; c < 2; ++c) {
          if (leader) tma_wait_group_read<1>();      // the reduce that last read this panel has finished reading
          named_bar_sync(1, 128);
          if (piece == 0 || row >= 64) {
            uint8_t* prow = sDq + buf * kDqPanelBytes + row * 128;
#pragma unroll
            for (int g = 0; g < 8; ++g)
              st_shared_v4(prow + ((g ^ (row & 7)) << 4), r[c][g * 4], r[c][g * 4 + 1], r[c][g * 4 + 2], r[c][g * 4 + 3]);
          }
          fence_proxy_async_smem();
          named_bar_sync(2, 128);
          if (leader) {
            if (piece == 0)
              tma_reduce_add_2d(&map_dq_a, sDq + buf * kDqPanelBytes, s * kSub + c * 32, bh * kDqk);
            else
              tma_reduce_add_2d(&map_dq_b, sDq + buf * kDqPanelBytes + 64 * 128, s * kSub + c * 32, bh * kDqk + 128);
            tma_commit_group();
          }
          buf ^= 1;
        }
      }
    }
    if (leader) tma_wait_group<0>();
    __syncwarp();
  } else {
    setmaxnreg_dec<kAuxRegs>();   // warps 14-15: release their registers
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 12) tmem_dealloc<512>(tmem);
}

// dq_acc^T [BH, 192, N] fp32 -> dq [BH, N, 192] bf16 (RN-even): 64 x 64 tiles through shared memory, reads coalesced
// along the queries, writes coalesced along the features.  qs != nullptr: the accumulator is int32 fixed point and query n
// of head bh carries the scale qs[bh * N + n] (deterministic mode).
__global__ void __launch_bounds__(256)
dq_transpose_convert_kernel(const float* __restrict__ acc, __nv_bfloat16* __restrict__ dq, int N, int n_pitch,
                            const float* __restrict__ qs) {
  // (acc rows are n_pitch floats apart: N rounded up to 128, so that a ragged N keeps the rows 16-byte aligned for TMA)
  __shared__ float tile[64][65];
  const int bh = blockIdx.z, f0 = blockIdx.y * 64, n0 = blockIdx.x * 64;
  const int tx = threadIdx.x & 63, ty = threadIdx.x >> 6;          // 64 x 4
  const float* src = acc + (static_cast<size_t>(bh) * kDqk + f0) * n_pitch + n0;
  const bool q_valid = n0 + tx < N;
  const float inv = qs && q_valid ? 1.0f / __ldg(qs + static_cast<size_t>(bh) * N + n0 + tx) : 1.0f;
#pragma unroll
  for (int r = ty; r < 64; r += 4) {                               // [feature][query]
    const float x = q_valid ? __ldcs(src + static_cast<size_t>(r) * n_pitch + tx) : 0.f;
    tile[r][tx] = qs ? static_cast<float>(__float_as_int(x)) * inv : x;
  }
  __syncthreads();
  __nv_bfloat16* dst = dq + (static_cast<size_t>(bh) * N + n0) * kDqk + f0;
#pragma unroll
  for (int r = ty; r < 64; r += 4)                                 // [query][feature]
    if (n0 + r < N) dst[static_cast<size_t>(r) * kDqk + tx] = __float2bfloat16_rn(tile[tx][r]);
}

}  // namespace

cudaError_t launch_attn_chunk_bwd_mla_sm100(const void* q, const void* k, const void* v, const void* dO,
                                            const float* lse2, const float* D, float* dq_acc_t, void* dk, void* dv,
                                            int BH, int N, int nk_stride, int k_off, int nk, float scale,
                                            const float* dq_qs, int dkv_dtype, cudaStream_t stream) {
  CUtensorMap mq, mk, mv, mdo, mdqa, mdqb;
  const CUtensorMapDataType dt = CU_TENSOR_MAP_DATA_TYPE_BFLOAT16;
  const CUtensorMapDataType dqt = dq_qs ? CU_TENSOR_MAP_DATA_TYPE_INT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32;
  const int n_stat = (N + 127) / 128 * 128;      // row stride of lse2, D and of the transposed dQ accumulator
  if (nk % kKeys && k_off + nk != nk_stride) return cudaErrorInvalidValue;   // only the head's last key tile may be ragged
  // dq_acc_t is [BH*192][n_stat] with N valid columns: the reduce-add clips the queries past the end
  if (!make_tmap_3d(&mq, q, dt, 2, BH, N, kDqk, kSub, 64, kSwizzle128B) ||
      !make_tmap_3d(&mk, k, dt, 2, BH, nk_stride, kDqk, kKeys, 64, kSwizzle128B) ||
      !make_tmap_3d(&mv, v, dt, 2, BH, nk_stride, kDv, kKeys, 64, kSwizzle128B) ||
      !make_tmap_3d(&mdo, dO, dt, 2, BH, N, kDv, kSub, 64, kSwizzle128B) ||
      !make_tmap_2d_pitched(&mdqa, dq_acc_t, dqt, 4, (uint64_t)BH * kDqk, N, n_stat, 128, 32, kSwizzle128B) ||
      !make_tmap_2d_pitched(&mdqb, dq_acc_t, dqt, 4, (uint64_t)BH * kDqk, N, n_stat, 64, 32, kSwizzle128B))
    return cudaErrorInvalidValue;
  auto kern = attn_chunk_bwd_mla_kernel;
  static unsigned char configured[kMaxDevices];
  if (cudaError_t e = set_max_dyn_smem_once(kern, kSmemBytes, configured); e != cudaSuccess) return e;
  dim3 grid((nk + kKeys - 1) / kKeys, BH);
  kern<<<grid, kThreads, kSmemBytes, stream>>>(mq, mk, mv, mdo, mdqa, mdqb, lse2, D, dk, dv, dkv_dtype == RINGX_F32, N, n_stat,
                                               nk_stride, k_off, scale * 1.4426950408889634f, scale, dq_qs);
  count_launch();
  return cudaGetLastError();
}

cudaError_t launch_dq_transpose_convert_mla(const float* dq_acc_t, void* dq, int BH, int N, const float* dq_qs,
                                            cudaStream_t stream) {
  dim3 grid((N + 63) / 64, kDqk / 64, BH);
  dq_transpose_convert_kernel<<<grid, 256, 0, stream>>>(dq_acc_t, static_cast<__nv_bfloat16*>(dq), N, (N + 127) / 128 * 128, dq_qs);
  return cudaGetLastError();
}

}  // namespace ringx
