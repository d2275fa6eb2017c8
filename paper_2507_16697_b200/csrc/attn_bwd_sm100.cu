// attn_bwd_sm100.cu -- one KV-chunk pass of the backward on tcgen05 tensor cores.
//
// A CTA owns one 128-key tile (K_j, V_j) of one head and loops over all 128-row query tiles i of that head:
//   S^T  = K_j Q_i^T                      P^T  = exp2(scale*log2e * S^T - lse2_i)   (P recomputed from the saved
//   dP^T = V_j dO_i^T                     dS^T = P^T o (dP^T - D_i)                  *global* LSE; reading g8)
//   dV_j += P^T dO_i      dK_j += dS^T Q_i      dQ_i += dS K_j                       (dS carries `scale`: phase B forms
// scale*dP - scale*D_i with one FFMA2).  dK_j, dV_j live in TMEM for the whole loop and are written once
// (atomic-free: the CTA owns the tile); dQ_i is reduce-added into the fp32 accumulator by TMA (cp.reduce.async.bulk) --
// the single-GPU image of "the gradient for Q is accumulated ... over N steps".
//
// Roles (512 threads):  warps 0-7  compute (thread = key row = TMEM lane; warps 0-3 take query columns 0-63 of the
//                                  tile, warps 4-7 columns 64-127)
//                       warps 8-11 dQ drain (thread = query row): TMEM -> registers (TMEM columns released at once)
//                                  -> swizzled fp32 staging panels -> TMA reduce-add into dq_acc
//                       warp  12   TMA producer (K_j,V_j once; then the Q_i/lse2_i/D_i and dO_i rings)
//                       warp  13   MMA issuer
//                       warps 14-15 idle (complete the fourth warpgroup for setmaxnreg)
// TMEM columns: S^T [0,128) (P^T, bf16, overwrites the first 32 columns of each 64-column half), dP^T [128,256),
// dV [256,256+d), dK [256+d,256+2d), dQ [384,448) for d = 64; for d = 128 dQ overlays dP^T (drained before the next
// dP^T is issued).  dS^T goes to shared memory as a [keys][queries] bf16 tile that serves as the K-major A operand of
// dK += dS^T Q and as the MN-major A operand of dQ = dS K.
// Pipeline: the compute warps alternate phase A (S^T -> P^T) and phase B (dP^T -> dS^T) while the tensor core runs
// {dV(i), S^T(i+1)} behind phase A and {dQ(i), dK(i), dP^T(i+1)} behind phase B (dQ first, so that its drain runs
// under the dK MMA); in-order MMA execution makes the P^T / S^T overlay safe.
#include <mutex>

#include "kernels.cuh"

namespace ringx {
namespace {

using namespace ptx;

__device__ unsigned g_bwd_smem_probe;   // written by the alignment probe launch (module memory: nothing is allocated)

constexpr int kTile = 128;
constexpr int kBwdThreads = 512;                 // 4 warpgroups; registers re-split with setmaxnreg
constexpr int kBwdComputeRegs = 176, kBwdDrainRegs = 96, kBwdAuxRegs = 40;   // 256*176 + 128*96 + 128*40 = 62464
// Which of the 16 element pairs per 32-column half of phase A take 2^x from the FMA-pipe polynomial (ptx::ex2_poly2)
// instead of MUFU.EX2.  At d = 64 phase A's 16 ex2 per clock are the co-limiter (5 MMAs of half the length per
// exponential): every fourth pair on the FMA pipe measured +4 % (C4 backward 897 -> 935 TFLOP/s); at d = 128 the
// tensor chain hides phase A and any share measured -1 %, so it stays on the MUFU.
constexpr unsigned kBwdPolyMaskD64 = 0x8888, kBwdPolyMaskD128 = 0x0000;

template <int kD>
struct BwdCfg {
  static constexpr int kPanels = kD / 64;
  static constexpr int kPanelBytes = 128 * 128;
  static constexpr int kTileBytes = kPanels * kPanelBytes;     // one [128, d] bf16 tile
  static constexpr int kQStages = kD == 64 ? 3 : 2;            // Q_i (+ lse2_i, D_i) ring: live from S^T(i) to dK(i)
  static constexpr int kDoStages = kD == 64 ? 3 : 1;           // dO_i ring: live from dP^T(i) to dV(i)
  static constexpr int kQStageBytes = kTileBytes + 1024;       // Q, lse2[128], D[128]
  static constexpr int kDsBytes = 2 * kPanelBytes;             // dS^T [128 keys][128 queries] bf16
  static constexpr int kDqPanelBytes = 128 * 128;              // dQ staging: [128 rows][32 fp32], 128B-swizzled
  static constexpr int kAlignSlack = kD == 64 ? 1024 : 0;      // d = 128 uses every byte: base must be 1 KB aligned
  static constexpr int kSmemBytes = kAlignSlack + 2 * kTileBytes + kQStages * kQStageBytes + kDoStages * kTileBytes +
                                    kDsBytes + 2 * kDqPanelBytes + 256;
  static constexpr uint32_t tS = 0, tDP = 128, tDV = 256, tDK = 256 + kD, tDQ = kD == 64 ? 384 : 128;
  static constexpr bool kDqOverlaysDp = kD != 64;
  // d = 64 leaves 64 TMEM columns: K_j and V_j (bf16, 32 columns each) are copied there once and serve as the A operands
  // of S^T = K Q^T and dP^T = V dO^T, and dS^T (bf16) is also written over the dP^T columns as the A operand of dK +=
  // dS^T Q.  The SM's shared memory (128 B/clk, which the SS MMAs saturate) then carries 64 KB less per step.
  static constexpr bool kTmemOperands = kD == 64;
  static constexpr uint32_t tK = 448, tV = 480;
  static constexpr unsigned kPolyMask = kD == 64 ? kBwdPolyMaskD64 : kBwdPolyMaskD128;
};

// Ragged sequences (N no multiple of 128).  Q_i, dO_i, K_j, V_j come through [BH][rows][d] tensor maps: rows past the end
// of a head read as zero, and the dQ reduce-add skips them.  lse2 / D are [BH][n_stat] with n_stat = N rounded up to 128
// and lse2 = +inf in the padding, so P = 0 for query rows that do not exist.  kTail: the launch contains the key tile
// that runs past the end of the head; its missing keys (K row zero: score 0) get P = 0 by a select in phase A and their
// dK, dV rows are not stored.  A separate instantiation: launches over full tiles carry none of it.
template <int kD, bool kTail>
__global__ void __launch_bounds__(kBwdThreads, 1)
attn_chunk_bwd_kernel(const __grid_constant__ CUtensorMap map_q, const __grid_constant__ CUtensorMap map_k,
                      const __grid_constant__ CUtensorMap map_v, const __grid_constant__ CUtensorMap map_do,
                      const __grid_constant__ CUtensorMap map_dq, const float* __restrict__ lse2,
                      const float* __restrict__ Dvec,
                      void* __restrict__ dk, void* __restrict__ dv, int dkv_f32, int N, int n_stat, int nk_stride, int k_off,
                      float scale_log2, float scale, const float* __restrict__ dq_qs, unsigned* __restrict__ smem_probe) {
  using Cfg = BwdCfg<kD>;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  // d = 128 uses every byte of the 227 KB, so it cannot round the base up: the launcher proves the alignment of this
  // kernel's dynamic shared memory once per device with a probe launch (smem_probe != nullptr: report and return) and
  // refuses to launch (RINGX_ERR_CUDA) if the base is not 1 KB aligned -- no trap, no abort.
  if (smem_probe) {
    if (threadIdx.x == 0 && blockIdx.x == 0 && blockIdx.y == 0) *smem_probe = smem_u32(smem_raw) & 1023u;
    return;
  }
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t* sK = smem;
  uint8_t* sV = smem + Cfg::kTileBytes;
  uint8_t* sQ = smem + 2 * Cfg::kTileBytes;                    // [kQStages] Q_i | lse2_i | D_i
  uint8_t* sDo = sQ + Cfg::kQStages * Cfg::kQStageBytes;       // [kDoStages] dO_i
  uint8_t* sDs = sDo + Cfg::kDoStages * Cfg::kTileBytes;
  uint8_t* sDq = sDs + Cfg::kDsBytes;                          // 2 staging panels for the dQ reduce-add
  uint64_t* bars = reinterpret_cast<uint64_t*>(sDq + 2 * Cfg::kDqPanelBytes);
  uint64_t* kv_full = bars;          // TMA -> MMA: K_j, V_j
  uint64_t* s_full = bars + 1;       // MMA -> compute: S^T(i)
  uint64_t* dp_full = bars + 2;      // MMA -> compute: dP^T(i)
  uint64_t* p_full = bars + 3;       // compute -> MMA: P^T(i) in TMEM, S^T(i) consumed            (8 arrivals: one per warp)
  uint64_t* ds_full = bars + 4;      // compute -> MMA: dS^T(i) in smem, dP^T(i) consumed          (8 arrivals)
  uint64_t* ds_empty = bars + 5;     // MMA -> compute: dK(i), dQ(i) have read dS^T(i)
  uint64_t* dq_full = bars + 6;      // MMA -> drain: dQ(i) in TMEM
  uint64_t* dq_empty = bars + 7;     // drain -> MMA: dQ(i) in registers                            (4 arrivals)
  uint64_t* dkv_full = bars + 8;     // MMA -> compute: dK_j, dV_j complete
  uint64_t* q_full = bars + 9;       // [kQStages] TMA -> MMA, compute
  uint64_t* q_empty = q_full + Cfg::kQStages;
  uint64_t* do_full = q_empty + Cfg::kQStages;     // [kDoStages]
  uint64_t* do_empty = do_full + Cfg::kDoStages;
  uint64_t* kv_tmem_full = do_empty + Cfg::kDoStages;   // compute -> MMA: K_j, V_j copied to TMEM     (256 arrivals)
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(kv_tmem_full + 1);

  const int warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0);
  const int lane = threadIdx.x & 31;
  const int bh = blockIdx.y;
  const int n_q = (N + kTile - 1) / kTile;
  const int q_row0 = bh * N;                                  // rows of this head in the flat [BH*N] arrays (dq_qs)
  const int s_row0 = bh * n_stat;                             // ... in lse2, D
  const int k_in = k_off + blockIdx.x * kTile;                // first key row of my tile within the head
  const int k_row0 = bh * nk_stride + k_in;                   // ... in the flat [BH*nk_stride, d] arrays dK, dV

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
    mbar_init(kv_tmem_full, 256);
    for (int i = 0; i < Cfg::kQStages; ++i) {
      mbar_init(&q_full[i], 1);
      mbar_init(&q_empty[i], 1);
    }
    for (int i = 0; i < Cfg::kDoStages; ++i) {
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
      prefetch_tmap(&map_dq);
    }
    tmem_alloc<512>(tmem_slot);
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_slot;

  if (warp == 12) {
    // ------------------------------------------------------------------ TMA producer
    setmaxnreg_dec<kBwdAuxRegs>();
    const bool leader = elect_one();
    const uint64_t pol_kv = policy_evict_first();
    const uint64_t pol_q = policy_evict_last();      // Q/dO tiles are re-read by every CTA of the head
    if (leader) {
      mbar_arrive_expect_tx(kv_full, 2 * Cfg::kTileBytes);
#pragma unroll
      for (int p = 0; p < Cfg::kPanels; ++p) {
        tma_load_3d(sK + p * Cfg::kPanelBytes, &map_k, kv_full, p * 64, k_in, bh, pol_kv);
        tma_load_3d(sV + p * Cfg::kPanelBytes, &map_v, kv_full, p * 64, k_in, bh, pol_kv);
      }
    }
    __syncwarp();
    auto load_q = [&](int i, int st) {
      if (leader) {
        uint8_t* dst = sQ + st * Cfg::kQStageBytes;
        mbar_arrive_expect_tx(&q_full[st], Cfg::kQStageBytes);
#pragma unroll
        for (int p = 0; p < Cfg::kPanels; ++p)
          tma_load_3d(dst + p * Cfg::kPanelBytes, &map_q, &q_full[st], p * 64, i * kTile, bh, pol_q);
        bulk_load_1d(dst + Cfg::kTileBytes, lse2 + s_row0 + i * kTile, 512, &q_full[st]);
        bulk_load_1d(dst + Cfg::kTileBytes + 512, Dvec + s_row0 + i * kTile, 512, &q_full[st]);
      }
      __syncwarp();
    };
    load_q(0, 0);
    int qs = Cfg::kQStages > 1 ? 1 : 0, qph = Cfg::kQStages > 1 ? 0 : 1, ds = 0, dph = 0;
    for (int i = 0; i < n_q; ++i) {
      // dO_i: its slot is free once dV(i - kDoStages) has read it
      mbar_wait_relaxed(&do_empty[ds], dph ^ 1);
      if (leader) {
        mbar_arrive_expect_tx(&do_full[ds], Cfg::kTileBytes);
#pragma unroll
        for (int p = 0; p < Cfg::kPanels; ++p)
          tma_load_3d(sDo + ds * Cfg::kTileBytes + p * Cfg::kPanelBytes, &map_do, &do_full[ds], p * 64, i * kTile, bh,
                      pol_q);
      }
      __syncwarp();
      if (++ds == Cfg::kDoStages) { ds = 0; dph ^= 1; }
      // Q_{i+1}: its slot is free once dK(i + 1 - kQStages) has read it
      if (i + 1 < n_q) {
        mbar_wait_relaxed(&q_empty[qs], qph ^ 1);
        load_q(i + 1, qs);
        if (++qs == Cfg::kQStages) { qs = 0; qph ^= 1; }
      }
    }
  } else if (warp == 13) {
    // ------------------------------------------------------------------ MMA issuer
    setmaxnreg_dec<kBwdAuxRegs>();
    const bool leader = elect_one();
    constexpr uint32_t idesc_st = make_idesc_bf16(kTile, kTile, 0, 0);   // K_j (K-major) x Q_i^T (K-major)
    constexpr uint32_t idesc_kn = make_idesc_bf16(kTile, kD, 0, 1);      // A K-major/TMEM x B MN-major -> [128, d]
    constexpr uint32_t idesc_mn = make_idesc_bf16(kTile, kD, 1, 1);      // A MN-major (dS from dS^T) x B MN-major
    const uint32_t k_addr = smem_u32(sK), v_addr = smem_u32(sV), ds_addr = smem_u32(sDs);
    const uint32_t q_base = smem_u32(sQ), do_base = smem_u32(sDo);
    auto kmajor = [](uint32_t base, int k) {   // K-step k of a K-major [128 rows][d or 128] tile (64-element panels)
      return make_smem_desc_sw128(base + (k >> 2) * Cfg::kPanelBytes + (k & 3) * 32, 16, 1024);
    };
    auto mnmajor = [](uint32_t base, int k) {  // K-step k (16 rows) of a [K rows][MN contiguous] tile
      return make_smem_desc_sw128(base + k * 2048, Cfg::kPanelBytes, 1024);
    };
    auto commit = [&](uint64_t* bar) {
      if (leader) mma_commit(bar);
      __syncwarp();
    };
    // S^T(i) = K_j Q_i^T ; dP^T(i) = V_j dO_i^T
    auto issue_st = [&](uint32_t q_addr) {
      if (leader) {
#pragma unroll
        for (int k = 0; k < kD / 16; ++k) {
          if (Cfg::kTmemOperands) mma_ts(tmem + Cfg::tS, tmem + Cfg::tK + k * 8, kmajor(q_addr, k), idesc_st, k > 0);
          else mma_ss(tmem + Cfg::tS, kmajor(k_addr, k), kmajor(q_addr, k), idesc_st, k > 0);
        }
        mma_commit(s_full);
      }
      __syncwarp();
    };
    auto issue_dpt = [&](uint32_t do_addr) {
      if (leader) {
#pragma unroll
        for (int k = 0; k < kD / 16; ++k) {
          if (Cfg::kTmemOperands) mma_ts(tmem + Cfg::tDP, tmem + Cfg::tV + k * 8, kmajor(do_addr, k), idesc_st, k > 0);
          else mma_ss(tmem + Cfg::tDP, kmajor(v_addr, k), kmajor(do_addr, k), idesc_st, k > 0);
        }
        mma_commit(dp_full);
      }
      __syncwarp();
    };
    mbar_wait(kv_full, 0);
    if (Cfg::kTmemOperands) mbar_wait(kv_tmem_full, 0);
    mbar_wait(&q_full[0], 0);
    tc_fence_after();
    issue_st(q_base);
    mbar_wait(&do_full[0], 0);
    tc_fence_after();
    issue_dpt(do_base);
    int qs = 0, qph = 0, ds = 0, dph = 0;
    for (int i = 0; i < n_q; ++i) {
      const uint32_t q_addr = q_base + qs * Cfg::kQStageBytes, do_addr = do_base + ds * Cfg::kTileBytes;
      const int cur_qs = qs, cur_ds = ds;
      if (++qs == Cfg::kQStages) { qs = 0; qph ^= 1; }
      if (++ds == Cfg::kDoStages) { ds = 0; dph ^= 1; }
      const bool more = i + 1 < n_q;
      // ---- behind phase A: dV += P^T(i) dO_i, then S^T(i+1)
      mbar_wait(p_full, i & 1);
      tc_fence_after();
      if (leader) {
#pragma unroll
        for (int k = 0; k < kTile / 16; ++k)
          mma_ts(tmem + Cfg::tDV, tmem + Cfg::tS + (k >> 2) * 64 + (k & 3) * 8, mnmajor(do_addr, k), idesc_kn,
                 i > 0 || k > 0);
        mma_commit(&do_empty[cur_ds]);
      }
      __syncwarp();
      if (more) {
        mbar_wait(&q_full[qs], qph);
        tc_fence_after();
        issue_st(q_base + qs * Cfg::kQStageBytes);
      }
      // ---- behind phase B: dQ(i) = dS(i) K_j (drained under the next MMA), dK += dS^T(i) Q_i, then dP^T(i+1)
      mbar_wait(ds_full, i & 1);
      if (!Cfg::kDqOverlaysDp && i > 0) mbar_wait(dq_empty, (i - 1) & 1);
      tc_fence_after();
      if (leader) {
#pragma unroll
        for (int k = 0; k < kTile / 16; ++k)
          mma_ss(tmem + Cfg::tDQ, mnmajor(ds_addr, k), mnmajor(k_addr, k), idesc_mn, k > 0);
        mma_commit(dq_full);
#pragma unroll
        for (int k = 0; k < kTile / 16; ++k)
          if (Cfg::kTmemOperands)
            mma_ts(tmem + Cfg::tDK, tmem + Cfg::tDP + (k >> 2) * 64 + (k & 3) * 8, mnmajor(q_addr, k), idesc_kn,
                   i > 0 || k > 0);
          else
            mma_ss(tmem + Cfg::tDK, kmajor(ds_addr, k), mnmajor(q_addr, k), idesc_kn, i > 0 || k > 0);
        mma_commit(ds_empty);
        mma_commit(&q_empty[cur_qs]);
      }
      __syncwarp();
      if (more) {
        mbar_wait(&do_full[ds], dph);
        if (Cfg::kDqOverlaysDp) mbar_wait(dq_empty, i & 1);   // dQ(i) sits in the dP^T columns until drained
        tc_fence_after();
        issue_dpt(do_base + ds * Cfg::kTileBytes);
      }
    }
    commit(dkv_full);
  } else if (warp < 8) {
    // ------------------------------------------------------------------ compute warps
    setmaxnreg_inc<kBwdComputeRegs>();
    const int half = warp >> 2;                                  // which 64 query columns of the tile
    const int row = (warp & 3) * 32 + lane;                      // key row of the tile = TMEM lane
    const uint32_t lane_off = static_cast<uint32_t>((warp & 3) * 32) << 16;
    const uint32_t tS = tmem + Cfg::tS + lane_off + half * 64;   // my S^T columns; P^T goes to the first 32 of them
    const uint32_t tDP = tmem + Cfg::tDP + lane_off + half * 64;
    uint8_t* ds_row = sDs + half * Cfg::kPanelBytes + row * 128;
    const float2 sc2 = make_float2(scale_log2, scale_log2);
    const float2 scl2 = make_float2(scale, scale);               // dS^T carries `scale` (Dvec holds scale * D_i)
    const bool key_valid = !kTail || k_in + row < nk_stride;
    if (Cfg::kTmemOperands) {
      // K_j (warps 0-3) / V_j (warps 4-7): my row of the 128B-swizzled tile -> my TMEM lane (2 bf16 per column)
      mbar_wait(kv_full, 0);
      const uint8_t* src = (half == 0 ? sK : sV) + row * 128;
      uint32_t kvr[32];
#pragma unroll
      for (int c = 0; c < 8; ++c) {
        const float4 x = ld_shared_v4(src + ((c ^ (row & 7)) << 4));
        kvr[c * 4 + 0] = __float_as_uint(x.x);
        kvr[c * 4 + 1] = __float_as_uint(x.y);
        kvr[c * 4 + 2] = __float_as_uint(x.z);
        kvr[c * 4 + 3] = __float_as_uint(x.w);
      }
      tmem_st_x32(tmem + (half == 0 ? Cfg::tK : Cfg::tV) + lane_off, kvr);
      tmem_wait_st();
      tc_fence_before();
      mbar_arrive(kv_tmem_full);
    }
    int stage = 0, phase = 0;
    for (int i = 0; i < n_q; ++i) {
      const float4* stats = reinterpret_cast<const float4*>(sQ + stage * Cfg::kQStageBytes + Cfg::kTileBytes);
      const float4* lse4 = stats + half * 16;                    // lse2 of my 64 query columns
      const float4* d4 = stats + 32 + half * 16;                 // D of my 64 query columns
      mbar_wait(&q_full[stage], phase);
      if (++stage == Cfg::kQStages) { stage = 0; phase ^= 1; }
      // ---- phase A: P^T = exp2(scale_log2 * S^T - lse2)
      // (lse2 / D are read from shared memory eight 16-byte loads at a time, ahead of the arithmetic that uses
      // them, so that their latency is paid once per half and mostly behind the mbarrier wait)
      float4 aux[8];
#pragma unroll
      for (int g = 0; g < 8; ++g) aux[g] = ld_shared_v4(lse4 + g);
      mbar_wait(s_full, i & 1);
      tc_fence_after();
      float2 p[32];
      {
        uint32_t s0[32], s1[32];
        tmem_ld_x32(tS, s0);
        tmem_ld_x32(tS + 32, s1);
        auto half_a = [&](const uint32_t (&s)[32], int c) {
          float2 x[16];
#pragma unroll
          for (int g = 0; g < 8; ++g) {
            x[g * 2] = ffma2(make_float2(__uint_as_float(s[g * 4 + 0]), __uint_as_float(s[g * 4 + 1])), sc2,
                             make_float2(-aux[g].x, -aux[g].y));
            x[g * 2 + 1] = ffma2(make_float2(__uint_as_float(s[g * 4 + 2]), __uint_as_float(s[g * 4 + 3])), sc2,
                                 make_float2(-aux[g].z, -aux[g].w));
          }
          if (c == 0) {
#pragma unroll
            for (int g = 0; g < 8; ++g) aux[g] = ld_shared_v4(lse4 + 8 + g);     // second half's lse2
          } else {
#pragma unroll
            for (int g = 0; g < 8; ++g) aux[g] = ld_shared_v4(d4 + g);           // phase B's first half of D
          }
          uint32_t pk[16];
#pragma unroll
          for (int e = 0; e < 16; ++e) {
            float2 pe = ((Cfg::kPolyMask >> e) & 1) ? ex2_poly2(x[e]) : make_float2(ex2(x[e].x), ex2(x[e].y));
            if (kTail && !key_valid) pe = make_float2(0.f, 0.f);       // a key past the end of the head
            p[c * 16 + e] = pe;
            pk[e] = pack_bf16x2(pe.x, pe.y);
          }
          tmem_st_x16(tS + c * 16, pk);      // overlays only S^T columns this thread has already loaded
        };
        tmem_wait_ld_x32(s0);
        tmem_wait_ld_x32(s1);
        half_a(s0, 0);
        half_a(s1, 1);
      }
      tmem_wait_st();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(p_full);          // one arrival per warp (8): 256 separate arrivals are 256 shared-memory atomics
      // ---- phase B: dS^T = P^T o (dP^T - D), bf16, to shared memory [keys][queries] (128B-swizzled rows)
      mbar_wait(dp_full, i & 1);
      if (i > 0) mbar_wait(ds_empty, (i - 1) & 1);
      tc_fence_after();
      {
        uint32_t dp0[32], dp1[32];
        tmem_ld_x32(tDP, dp0);
        tmem_ld_x32(tDP + 32, dp1);
        auto half_b = [&](const uint32_t (&dp)[32], int c) {
          float2 t[16];
          uint32_t dsk[16];
#pragma unroll
          for (int g = 0; g < 8; ++g) {
            t[g * 2] = ffma2(make_float2(__uint_as_float(dp[g * 4 + 0]), __uint_as_float(dp[g * 4 + 1])), scl2,
                             make_float2(-aux[g].x, -aux[g].y));
            t[g * 2 + 1] = ffma2(make_float2(__uint_as_float(dp[g * 4 + 2]), __uint_as_float(dp[g * 4 + 3])), scl2,
                                 make_float2(-aux[g].z, -aux[g].w));
          }
          if (c == 0) {
#pragma unroll
            for (int g = 0; g < 8; ++g) aux[g] = ld_shared_v4(d4 + 8 + g);       // second half of D
          }
#pragma unroll
          for (int g = 0; g < 4; ++g) {     // 8 queries = one 16-byte chunk of the row
            const int e = g * 4;
            const float2 w0 = fmul2(p[c * 16 + e + 0], t[e + 0]), w1 = fmul2(p[c * 16 + e + 1], t[e + 1]);
            const float2 w2 = fmul2(p[c * 16 + e + 2], t[e + 2]), w3 = fmul2(p[c * 16 + e + 3], t[e + 3]);
            const int chunk = c * 4 + g;
            const uint32_t u0 = pack_bf16x2(w0.x, w0.y), u1 = pack_bf16x2(w1.x, w1.y);
            const uint32_t u2 = pack_bf16x2(w2.x, w2.y), u3 = pack_bf16x2(w3.x, w3.y);
            st_shared_v4(ds_row + ((chunk ^ (row & 7)) << 4), u0, u1, u2, u3);
            if (Cfg::kTmemOperands) { dsk[g * 4 + 0] = u0; dsk[g * 4 + 1] = u1; dsk[g * 4 + 2] = u2; dsk[g * 4 + 3] = u3; }
          }
          // (overlays only dP^T columns this thread has already loaded; dP^T(i+1) is issued behind dK(i))
          if (Cfg::kTmemOperands) tmem_st_x16(tDP + c * 16, dsk);
        };
        tmem_wait_ld_x32(dp0);
        tmem_wait_ld_x32(dp1);
        half_b(dp0, 0);
        half_b(dp1, 1);
      }
      fence_proxy_async_smem();
      if (Cfg::kTmemOperands) tmem_wait_st();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(ds_full);
    }
    // ---- epilogue: dV_j (warps 0-3) and dK_j (warps 4-7), bf16, written once
    mbar_wait(dkv_full, 0);
    tc_fence_after();
    const uint32_t tSrc = tmem + (half == 0 ? Cfg::tDV : Cfg::tDK) + lane_off;
    const size_t out_off = (static_cast<size_t>(k_row0) + row) * kD;
    // bf16 (the single-device result), or fp32 (one device's share of a cross-device sum: RingX_a/b reduce the shares
    // in fp32 and round once, instead of rounding every share to bf16 first)
#pragma unroll
    for (int c = 0; c < kD / 32; ++c) {
      uint32_t r[32];
      tmem_ld_x32(tSrc + c * 32, r);
      tmem_wait_ld();
      if (!key_valid) continue;              // (after the warp-wide TMEM load) a key row past the end of the head
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
    // ------------------------------------------------------------------ dQ drain warps (8-11)
    // TMEM -> registers (all d columns at once, so the TMEM columns go back to the MMA warp immediately)
    // -> 128B-swizzled fp32 staging panel [128 rows][32 cols] -> one TMA reduce-add per panel
    // (cp.reduce.async.bulk.tensor ... .add): full-line L2 atomics issued by the TMA engine, nothing on the LSU
    // but conflict-free 16-byte shared stores.
    setmaxnreg_dec<kBwdDrainRegs>();
    const int row = (warp & 3) * 32 + lane;                      // query row of the tile = TMEM lane
    const uint32_t tDQ = tmem + Cfg::tDQ + (static_cast<uint32_t>((warp & 3) * 32) << 16);
    const bool leader = warp == 8 && elect_one();
    // Deterministic mode (dq_qs != nullptr): dq_acc is an int32 fixed-point accumulator.  Row r of the head carries a
    // scale dq_qs[r] chosen from a bound on |dQ_r| (launch_dq_fixed_scale), every fp32 partial is scaled and rounded
    // to an integer here, and the TMA reduce-adds are integer adds: associative, so the sum does
    // not depend on the order in which the CTAs' adds arrive -- bit-reproducible dQ with no ordering between CTAs.
    const bool fixed = dq_qs != nullptr;
    const float* qs_row = fixed ? dq_qs + q_row0 + row : nullptr;
    float qs_next = fixed && row < N ? __ldg(qs_row) : 1.f;
    int buf = 0;
    for (int i = 0; i < n_q; ++i) {
      const float qs = qs_next;
      if (fixed && (i + 1) * kTile + row < N) qs_next = __ldg(qs_row + (i + 1) * kTile);   // ahead of the wait: latency hidden
      mbar_wait(dq_full, i & 1);
      tc_fence_after();

#pragma unroll
      for (int rd = 0; rd < kD / 64; ++rd) {     // 64 columns per round keep the drain warps under 100 registers
        uint32_t r[2][32];
#pragma unroll
        for (int c = 0; c < 2; ++c) tmem_ld_x32(tDQ + rd * 64 + c * 32, r[c]);
#pragma unroll
        for (int c = 0; c < 2; ++c) tmem_wait_ld_x32(r[c]);
        if (rd == kD / 64 - 1) {
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(dq_empty);   // the whole dQ(i) tile has left TMEM: hand the columns back
        }
        if (fixed) {
#pragma unroll
          for (int c = 0; c < 2; ++c)
#pragma unroll
            for (int e = 0; e < 32; ++e)
              r[c][e] = static_cast<uint32_t>(__float2int_rn(__uint_as_float(r[c][e]) * qs));
        }
#pragma unroll
        for (int c = 0; c < 2; ++c) {
          if (leader) tma_wait_group_read<1>();      // the reduce that last read this panel has finished reading
          named_bar_sync(1, 128);
          uint8_t* prow = sDq + buf * Cfg::kDqPanelBytes + row * 128;
#pragma unroll
          for (int g = 0; g < 8; ++g)
            st_shared_v4(prow + ((g ^ (row & 7)) << 4), r[c][g * 4], r[c][g * 4 + 1], r[c][g * 4 + 2], r[c][g * 4 + 3]);
          fence_proxy_async_smem();
          named_bar_sync(2, 128);
          if (leader) {
            tma_reduce_add_3d(&map_dq, sDq + buf * Cfg::kDqPanelBytes, rd * 64 + c * 32, i * kTile, bh);
            tma_commit_group();
          }
          buf ^= 1;
        }
      }
    }
    if (leader) tma_wait_group<0>();
    __syncwarp();
  } else {
    setmaxnreg_dec<kBwdAuxRegs>();   // warps 14-15: release their registers
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 12) tmem_dealloc<512>(tmem);
}

template <int kD, bool kTail>
cudaError_t launch_tt(const CUtensorMap& mq, const CUtensorMap& mk, const CUtensorMap& mv, const CUtensorMap& mdo,
                      const CUtensorMap& mdq, const float* lse2, const float* D, void* dk, void* dv, int dkv_f32, int BH,
                      int N, int n_stat, int nk_stride, int k_off, int nk, float scale, const float* dq_qs,
                      cudaStream_t stream) {
  using Cfg = BwdCfg<kD>;
  auto kern = attn_chunk_bwd_kernel<kD, kTail>;
  static unsigned char configured[kMaxDevices];
  // First use on a device (kernels without alignment slack, d = 128): prove that the dynamic shared memory of this kernel
  // starts 1 KB aligned (see the kernel).  The probe runs on a stream of its own that exists only for this check (a host
  // object, no device memory) and the host waits for THAT stream: the caller's stream is neither used nor synchronised.
  // A caller's stream that is being captured is refused before this launcher touches anything (the first backward on a
  // device belongs outside a capture).
  static unsigned char probed[kMaxDevices];    // 0 = not yet, 1 = aligned, 2 = misaligned; guarded by probe_mu
  static std::mutex probe_mu;
  int dev = 0;
  bool need_probe = false, cacheable = false;
  if (Cfg::kAlignSlack == 0) {
    if (cudaError_t e = cudaGetDevice(&dev); e != cudaSuccess) return e;
    cacheable = dev >= 0 && dev < kMaxDevices;
    {
      std::lock_guard<std::mutex> guard(probe_mu);
      if (cacheable && probed[dev] == 2) return cudaErrorInvalidConfiguration;
      need_probe = !cacheable || !probed[dev];
    }
    if (need_probe) {
      cudaStreamCaptureStatus capturing = cudaStreamCaptureStatusNone;
      if (cudaError_t e = cudaStreamIsCapturing(stream, &capturing); e != cudaSuccess) return e;
      if (capturing != cudaStreamCaptureStatusNone) return cudaErrorStreamCaptureUnsupported;
    }
  }
  if (cudaError_t e = set_max_dyn_smem_once(kern, Cfg::kSmemBytes, configured); e != cudaSuccess) return e;
  if (need_probe) {
    std::lock_guard<std::mutex> guard(probe_mu);
    if (!cacheable || !probed[dev]) {          // (another thread may have probed this device in the meantime)
      unsigned* flag = nullptr;
      unsigned h = 0xffffffffu;
      cudaError_t e = cudaGetSymbolAddress(reinterpret_cast<void**>(&flag), g_bwd_smem_probe);
      if (e != cudaSuccess) return e;
      cudaStream_t probe_stream = nullptr;
      if ((e = cudaStreamCreateWithFlags(&probe_stream, cudaStreamNonBlocking)) != cudaSuccess) return e;
      kern<<<1, 32, Cfg::kSmemBytes, probe_stream>>>(mq, mk, mv, mdo, mdq, nullptr, nullptr, nullptr, nullptr, 0, 0, 0, 0, 0,
                                                     0.f, 0.f, nullptr, flag);
      e = cudaGetLastError();
      if (e == cudaSuccess) e = cudaMemcpyAsync(&h, flag, sizeof(h), cudaMemcpyDeviceToHost, probe_stream);
      if (e == cudaSuccess) e = cudaStreamSynchronize(probe_stream);
      cudaStreamDestroy(probe_stream);
      if (e != cudaSuccess) return e;
      if (cacheable) probed[dev] = h == 0 ? 1 : 2;
      if (h != 0) return cudaErrorInvalidConfiguration;
    } else if (probed[dev] == 2) {
      return cudaErrorInvalidConfiguration;
    }
  }
  dim3 grid((nk + kTile - 1) / kTile, BH);
  kern<<<grid, kBwdThreads, Cfg::kSmemBytes, stream>>>(mq, mk, mv, mdo, mdq, lse2, D, dk, dv, dkv_f32, N, n_stat, nk_stride,
                                                       k_off, scale * 1.4426950408889634f, scale, dq_qs, nullptr);
  count_launch();
  return cudaGetLastError();
}

template <int kD>
cudaError_t launch_t(const CUtensorMap& mq, const CUtensorMap& mk, const CUtensorMap& mv, const CUtensorMap& mdo,
                     const CUtensorMap& mdq, const float* lse2, const float* D, void* dk, void* dv, int dkv_f32, int BH,
                     int N, int n_stat, int nk_stride, int k_off, int nk, float scale, const float* dq_qs,
                     cudaStream_t stream) {
  if (nk % kTile)
    return launch_tt<kD, true>(mq, mk, mv, mdo, mdq, lse2, D, dk, dv, dkv_f32, BH, N, n_stat, nk_stride, k_off, nk, scale, dq_qs,
                               stream);
  return launch_tt<kD, false>(mq, mk, mv, mdo, mdq, lse2, D, dk, dv, dkv_f32, BH, N, n_stat, nk_stride, k_off, nk, scale, dq_qs,
                              stream);
}

}  // namespace

cudaError_t launch_attn_chunk_bwd_sm100(const void* q, const void* k, const void* v, const void* dO, const float* lse2,
                                        const float* D, float* dq_acc, void* dk, void* dv, int BH, int N,
                                        int nk_stride, int k_off, int nk, int d, float scale, const float* dq_qs,
                                        int dkv_dtype, cudaStream_t stream) {
  if (nk % kTile && k_off + nk != nk_stride) return cudaErrorInvalidValue;   // only the head's last key tile may be ragged
  CUtensorMap mq, mk, mv, mdo, mdq;
  const int dkv_f32 = dkv_dtype == RINGX_F32;
  const int n_stat = (N + kTile - 1) / kTile * kTile;      // row stride of lse2, D (launch_bwd_preprocess)
  const CUtensorMapDataType dt = CU_TENSOR_MAP_DATA_TYPE_BFLOAT16;
  // [BH][rows][d] views: tiles that run past the end of a head read zeros there, and the dQ reduce-add skips those rows
  if (!make_tmap_3d(&mq, q, dt, 2, BH, N, d, 128, 64, kSwizzle128B) ||
      !make_tmap_3d(&mk, k, dt, 2, BH, nk_stride, d, 128, 64, kSwizzle128B) ||
      !make_tmap_3d(&mv, v, dt, 2, BH, nk_stride, d, 128, 64, kSwizzle128B) ||
      !make_tmap_3d(&mdo, dO, dt, 2, BH, N, d, 128, 64, kSwizzle128B) ||
      !make_tmap_3d(&mdq, dq_acc, dq_qs ? CU_TENSOR_MAP_DATA_TYPE_INT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, BH, N, d, 128, 32,
                    kSwizzle128B))
    return cudaErrorInvalidValue;
  if (d == 64)
    return launch_t<64>(mq, mk, mv, mdo, mdq, lse2, D, dk, dv, dkv_f32, BH, N, n_stat, nk_stride, k_off, nk, scale, dq_qs, stream);
  return launch_t<128>(mq, mk, mv, mdo, mdq, lse2, D, dk, dv, dkv_f32, BH, N, n_stat, nk_stride, k_off, nk, scale, dq_qs, stream);
}

}  // namespace ringx
