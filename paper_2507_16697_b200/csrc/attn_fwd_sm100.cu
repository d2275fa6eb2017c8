// attn_fwd_sm100.cu -- one KV-chunk pass of the forward on tcgen05 tensor cores.
//
// For every query row of a [128 x 2]-row CTA tile and the keys [k_off, k_off + nk) of its head:
//   loc_out = softmax(scale q K_c^T) V_c,  loc_lse = log sum_j exp(scale q.k_j)      (Eq. 1/3/4)
// bf16 operands, fp32 accumulation ("mixed float32-bfloat16").
//
// Structure (one CTA per SM, 384 threads = 3 warpgroups; registers re-split with setmaxnreg):
//   warps 0-3   softmax warpgroup of query tile 0 (thread = one query row; owns TMEM lane = row)   224 regs
//   warps 4-7   softmax warpgroup of query tile 1                                                  224 regs
//   warp  8     TMA producer: Q tiles once, then the K/V ring (K_0, V_0, K_1, V_1, ...)              56 regs
//   warp  9     MMA issuer (one elected lane): S_t = Q_t K_j^T (SS), O_t += P_t V_j (P from TMEM)    56 regs
//   warps 10-11 idle (they only complete the third warpgroup so that setmaxnreg can be used)
// TMEM columns (d = 128): S_0 [0,128) S_1 [128,256) O_0 [256,384) O_1 [384,512); P_t (bf16) overwrites
// the first 64 columns of S_t.  The two query tiles ping-pong: while warpgroup t turns S_t into P_t the
// tensor core works on tile 1-t.  The MMA pipe executes in issue order, so S_t(j+1) -- issued right after
// O_t += P_t(j) V_j -- cannot overwrite P_t(j) early, and the commit that signals S_t(j+1) also proves
// O_t(j) complete: the softmax warps may rescale O_t in place without a further barrier.
// d = 64 has 128 TMEM columns to spare and uses them for a third score buffer: S number n = 2j + t goes to
// buffer n % 3 [0,384), O_0 [384,448), O_1 [448,512), and is issued behind PV number n - 3, i.e. one tile
// ahead, so a softmax warpgroup finds its next scores waiting (ring order K_0 K_1 V_0 K_2 V_1 ...).  Running
// ahead of PV_t(j-1) costs two waits on pv_done[t]: before the (rare) in-place rescale of O_t, and before P_t(j)
// is signalled (so that p_full cannot complete twice before the MMA warp has seen it once).
// Online softmax in the exp2 domain with a lazy running max (O, l are only rescaled when the row max
// grew by more than 2^8), so the rescale is off the common path.  The softmax streams S out of TMEM in
// 32-column pieces (the row max of piece c is taken while piece c+1 is in flight), uses the packed
// FFMA2/FADD2 and three-input FMNMX3 forms, and hands P to the tensor core in two 64-key halves so that
// the first half of O += P V starts while the second half of P is still being exponentiated.
#include "kernels.cuh"

namespace ringx {
namespace {

using namespace ptx;

constexpr int kBlockM = 128;          // query rows per tile (= TMEM lanes)
constexpr int kBlockN = 128;          // keys per KV tile
#ifndef RINGX_FWD_COLSPLIT_D64
#define RINGX_FWD_COLSPLIT_D64 1
#endif
#ifndef RINGX_FWD_COLSPLIT_D128
#define RINGX_FWD_COLSPLIT_D128 0
#endif
constexpr float kRescaleThreshold = 8.0f;   // log2 units
// d = 64 is bound by the softmax warps (one exponential per 4*64 tensor FLOPs: 2048 clk of MUFU.EX2 against 1024 clk
// of MMA per 128-key iteration).  Of the 16 element pairs of every 32-key piece, those in this mask take 2^x from the
// FMA-pipe polynomial ptx::ex2_poly2 (degree 4, relative error 2.7e-6: P also feeds the fp32 row sum behind LSE).
// Measured on C4 forward with three score buffers: 0 -> 781, 1/8 -> 796, 1/4 -> 791 TFLOP/s (the warps are close to
// issue-bound as well).  d = 128 is balanced and power-capped: it stays on the MUFU.
#ifndef RINGX_FWD_POLY_MASK_D64
#define RINGX_FWD_POLY_MASK_D64 0x8080
#endif
#ifndef RINGX_FWD_POLY_DEGREE
#define RINGX_FWD_POLY_DEGREE 4
#endif

template <int kD>
struct FwdCfg {
  static constexpr int kPanels = kD / 64;                    // 64 bf16 = one 128-byte swizzle row
  static constexpr int kPanelBytes = 128 * 128;              // 128 rows x 128 B
  static constexpr int kTileBytes = kPanels * kPanelBytes;   // Q, K or V tile
  static constexpr int kStages = kD == 128 ? 5 : 8;          // K/V ring slots
  static constexpr unsigned kPolyMask = kD == 64 ? RINGX_FWD_POLY_MASK_D64 : 0u;
  // Score buffers in TMEM.  d = 128: one per query tile (2 x 128 + 2 x 128 O columns = 512).  d = 64 leaves 128
  // columns, enough for a third buffer: the score MMAs then run one tile ahead (S number n = 2j + t goes to buffer
  // n % 3 and is issued behind PV number n - 3), so a softmax warpgroup never waits for its next scores.
  static constexpr int kSBufs = kD == 128 ? 2 : 3;
  static constexpr uint32_t kOBase = kSBufs * 128;           // O_t at kOBase + t * kD
  static constexpr int kBarBytes = 256;
  // Column split: the 128 keys of a score tile are shared by TWO softmax warpgroups (64 keys each), i.e. four softmax
  // warpgroups per CTA and four warps per scheduler instead of two -- the MUFU pipe then stays busy while other warps
  // are in their TMEM-load / row-max phase or wait on a barrier.  The two halves of a row exchange their row maxima
  // (and, in the epilogue, their row sums) through shared memory.
  static constexpr bool kColSplit = kD == 64 ? (RINGX_FWD_COLSPLIT_D64 != 0) : (RINGX_FWD_COLSPLIT_D128 != 0);
  static constexpr int kSoftmaxWarps = kColSplit ? 16 : 8;
  static constexpr int kProducerWarp = kSoftmaxWarps, kMmaWarp = kSoftmaxWarps + 1;
  static constexpr int kThreads = (kSoftmaxWarps + 4) * 32;
  // setmaxnreg moves registers inside the CTA's own pool (threads x the launch-time count: 384 x 168 / 640 x 96), so what
  // the softmax warpgroups gain must equal what the last warpgroup gives up: 256 x (224-168) = 128 x (168-56);
  // 512 x (112-96) = 128 x (96-32)
  static constexpr int kSoftmaxRegs = kColSplit ? 112 : 224;
  static constexpr int kAuxRegs = kColSplit ? 32 : 56;
  static constexpr int kXchBytes = kColSplit ? 2 * 2 * 2 * 128 * 4 : 0;    // [tile][parity][half][row] floats
  static constexpr int kSmemBytes = 1024 + 2 * kTileBytes + kStages * kTileBytes + kBarBytes + kXchBytes;
};

// Epilogue modes (kEpi): what happens to (loc_out, loc_lse) of this chunk
//   kEpiPartial   written as they are, fp32                       (first pass; ringx_attn_chunk_fwd)
//   kEpiFinal     loc_out written as bf16                         (single pass: the chunk is the whole sequence)
//   kEpiFold      folded into the running (o_acc, lse_acc) with the two-operand Eq. 5, in place, fp32
//   kEpiFoldFinal folded with (o_acc, lse_acc) and written to (o_out, lse_out) as bf16 (last pass)
// Folding here instead of in a separate lse_merge launch saves the round trip of loc_out through HBM; it is the same
// arithmetic as merge.cu's lse_merge_kernel, row by row (a thread owns a query row).
enum { kEpiPartial = 0, kEpiFinal = 1, kEpiFold = 2, kEpiFoldFinal = 3 };

template <int kD, int kEpi>
__global__ void __launch_bounds__(FwdCfg<kD>::kThreads, 1)
attn_chunk_fwd_kernel(const __grid_constant__ CUtensorMap map_q, const __grid_constant__ CUtensorMap map_k,
                      const __grid_constant__ CUtensorMap map_v, void* o_out, float* lse_out, const float* o_acc,
                      const float* lse_acc, int Nq, int nk_stride, int k_off, int n_kv, float scale_log2) {
  using Cfg = FwdCfg<kD>;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t* sQ = smem;
  uint8_t* sKV = smem + 2 * Cfg::kTileBytes;
  uint64_t* bars = reinterpret_cast<uint64_t*>(sKV + Cfg::kStages * Cfg::kTileBytes);
  uint64_t* q_full = bars;                  // [2]  TMA -> MMA
  uint64_t* s_full = bars + 2;              // [kSBufs] MMA -> softmax: score buffer b holds S number n (n % kSBufs == b)
  uint64_t* p_full = bars + 5;              // [2][2] softmax -> MMA: half h (64 keys) of P_t(j) in TMEM (O_t rescaled if needed)
  uint64_t* o_full = bars + 9;              // [2]  MMA -> softmax: last O_t complete
  uint64_t* pv_done = bars + 11;            // [2]  MMA -> softmax: O_t += P_t(j) V_j complete (used when kSBufs > 2)
  uint64_t* kv_full = bars + 13;            // [kStages]
  uint64_t* kv_empty = bars + 13 + Cfg::kStages;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 13 + 2 * Cfg::kStages);
  float* xch = reinterpret_cast<float*>(reinterpret_cast<uint8_t*>(bars) + Cfg::kBarBytes);   // column-split exchange

  const int warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0);   // provably warp-uniform: keeps MMA/TMA operands in uniform registers
  const int lane = threadIdx.x & 31;
  const int bh = blockIdx.y;
  const int q_row0 = bh * Nq + blockIdx.x * (2 * kBlockM);     // row in the [BH*Nq, d] view
  const int k_row0 = bh * nk_stride + k_off + blockIdx.z * n_kv * kBlockN;   // blockIdx.z = key split (split-KV)

  if (threadIdx.x == 0) {
    for (int i = 0; i < 2; ++i) {
      mbar_init(&q_full[i], 1);
      mbar_init(&p_full[2 * i], kBlockM);
      mbar_init(&p_full[2 * i + 1], kBlockM);
      mbar_init(&o_full[i], 1);
      mbar_init(&pv_done[i], 1);
    }
    for (int i = 0; i < Cfg::kSBufs; ++i) mbar_init(&s_full[i], 1);
    for (int i = 0; i < Cfg::kStages; ++i) {
      mbar_init(&kv_full[i], 1);
      mbar_init(&kv_empty[i], 1);
    }
    fence_mbar_init();
  }
  if (warp == Cfg::kProducerWarp) {
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

  if (warp == Cfg::kProducerWarp) {
    setmaxnreg_dec<Cfg::kAuxRegs>();
    // ------------------------------------------------------------------ TMA producer
    // (the whole warp runs the loop so that every operand is warp-uniform; one elected lane issues)
    {
      const bool leader = elect_one();
      const uint64_t pol_q = policy_evict_first();
      const uint64_t pol_kv = policy_evict_last();
      auto load_tile = [&](uint8_t* dst, const CUtensorMap* map, uint64_t* bar, int row, uint64_t pol) {
        if (leader) {
          mbar_arrive_expect_tx(bar, Cfg::kTileBytes);
#pragma unroll
          for (int p = 0; p < Cfg::kPanels; ++p) tma_load_2d(dst + p * Cfg::kPanelBytes, map, bar, p * 64, row, pol);
        }
        __syncwarp();
      };
      load_tile(sQ, &map_q, &q_full[0], q_row0, pol_q);
      // ring order = the order in which the MMA warp first touches the tiles: the K tiles of the kSBufs score MMAs
      // of the prologue, then per PV number n its V tile (n even) and the K tile of S number n + kSBufs (if even)
      //   kSBufs = 2: K_0 V_0 K_1 V_1 ...        kSBufs = 3: K_0 K_1 V_0 K_2 V_1 K_3 ...
      int stage = 0, phase = 0, loaded = 0;
      auto push = [&](const CUtensorMap* map, int j) {
        mbar_wait_relaxed(&kv_empty[stage], phase ^ 1);
        load_tile(sKV + stage * Cfg::kTileBytes, map, &kv_full[stage], k_row0 + j * kBlockN, pol_kv);
        if (loaded++ == 0) load_tile(sQ + Cfg::kTileBytes, &map_q, &q_full[1], q_row0 + kBlockM, pol_q);
        if (++stage == Cfg::kStages) { stage = 0; phase ^= 1; }
      };
      const int n_s = 2 * n_kv;                  // score / PV MMAs are numbered n = 2 j + t
      for (int m = 0; m < Cfg::kSBufs && m < n_s; m += 2) push(&map_k, m >> 1);
      for (int n = 0; n < n_s; n += 2) {
        push(&map_v, n >> 1);
        const int m = n + Cfg::kSBufs + (Cfg::kSBufs & 1);     // the even S number among n + kSBufs, n + 1 + kSBufs
        if (m < n_s) push(&map_k, m >> 1);
      }
    }
  } else if (warp == Cfg::kMmaWarp) {
    // ------------------------------------------------------------------ MMA issuer
    setmaxnreg_dec<Cfg::kAuxRegs>();
    {
      const bool leader = elect_one();
      constexpr uint32_t idesc_s = make_idesc_bf16(kBlockM, kBlockN, 0, 0);    // Q (K-major) x K^T (K-major)
      constexpr uint32_t idesc_o = make_idesc_bf16(kBlockM, kD, 0, 1);         // P (TMEM) x V (MN-major)
      const uint32_t q_addr = smem_u32(sQ), kv_addr = smem_u32(sKV);
      int stage = 0, phase = 0;
      auto advance = [&]() { if (++stage == Cfg::kStages) { stage = 0; phase ^= 1; } };
      // S number n (tile t = n & 1) = Q_t K^T from the K tile in ring slot `st`, into score buffer n % kSBufs
      auto issue_s = [&](int n, int t, int st) {
        const int buf = Cfg::kSBufs == 2 ? t : n % Cfg::kSBufs;
        const uint32_t a0 = q_addr + t * Cfg::kTileBytes, b0 = kv_addr + st * Cfg::kTileBytes;
        if (leader) {
#pragma unroll
          for (int k = 0; k < kD / 16; ++k) {
            const uint32_t off = (k >> 2) * Cfg::kPanelBytes + (k & 3) * 32;
            mma_ss(tmem + buf * kBlockN, make_smem_desc_sw128(a0 + off, 16, 1024),
                   make_smem_desc_sw128(b0 + off, 16, 1024), idesc_s, k > 0);
          }
          mma_commit(&s_full[buf]);
        }
        __syncwarp();
      };
      // O_t (+)= P V: keys [64*half, 64*half + 64) of PV number n (P sits in score buffer n % kSBufs)
      auto issue_o = [&](int n, int t, int st, int half, bool accumulate) {
        const int buf = Cfg::kSBufs == 2 ? t : n % Cfg::kSBufs;
        const uint32_t b0 = kv_addr + st * Cfg::kTileBytes;
        if (leader) {
#pragma unroll
          for (int k = half * 4; k < half * 4 + 4; ++k)
            mma_ts(tmem + Cfg::kOBase + t * kD, tmem + buf * kBlockN + k * 8,
                   make_smem_desc_sw128(b0 + k * 2048, Cfg::kPanelBytes, 1024), idesc_o, accumulate || k > 0);
        }
        __syncwarp();
      };
      auto commit = [&](uint64_t* bar) {
        if (leader) mma_commit(bar);
        __syncwarp();
      };
      // ring slots are taken in the producer's order; a K tile serves S numbers 2j, 2j+1, a V tile PV numbers 2j, 2j+1
      int k_slot = 0, v_slot = 0;
      auto acquire = [&]() {
        const int st = stage;
        mbar_wait(&kv_full[stage], phase);
        tc_fence_after();
        advance();
        return st;
      };
      auto score = [&](int m, int t) {   // issue S number m (tile t = m & 1); the odd one releases the K tile
        if (t == 0) k_slot = acquire();
        if (m < 2) {
          mbar_wait(&q_full[t], 0);
          tc_fence_after();
        }
        issue_s(m, t, k_slot);
        if (t == 1) commit(&kv_empty[k_slot]);
      };
      const int n_s = 2 * n_kv;
#pragma unroll
      for (int m = 0; m < Cfg::kSBufs; ++m)                            // prologue: the first kSBufs score tiles
        if (m < n_s) score(m, m & 1);
      for (int j = 0; j < n_kv; ++j) {
#pragma unroll
        for (int t = 0; t < 2; ++t) {
          const int n = 2 * j + t;
          if (t == 0) v_slot = acquire();
          mbar_wait(&p_full[2 * t], j & 1);
          tc_fence_after();
          issue_o(n, t, v_slot, 0, j > 0);
          mbar_wait(&p_full[2 * t + 1], j & 1);
          tc_fence_after();
          issue_o(n, t, v_slot, 1, true);
          if (Cfg::kSBufs > 2) commit(&pv_done[t]);
          if (t == 1) commit(&kv_empty[v_slot]);
          if (j + 1 == n_kv) commit(&o_full[t]);                              // last PV of tile t
          if (n + Cfg::kSBufs < n_s) score(n + Cfg::kSBufs, (t + Cfg::kSBufs) & 1);   // refill the buffer PV number n freed
        }
      }
    }
  } else if (warp < Cfg::kSoftmaxWarps) {
    // ------------------------------------------------------------------ softmax warpgroups
    setmaxnreg_inc<Cfg::kSoftmaxRegs>();
    const int t = Cfg::kColSplit ? warp >> 3 : warp >> 2;      // query tile
    const int hh = Cfg::kColSplit ? (warp >> 2) & 1 : 0;       // column split: which 64 keys of every score tile
    const uint32_t lane_off = static_cast<uint32_t>((warp & 3) * 32) << 16;
    const uint32_t tO = tmem + Cfg::kOBase + t * kD + lane_off;
    constexpr bool kFold = kEpi == kEpiFold || kEpi == kEpiFoldFinal;
    constexpr bool kOutBf16 = kEpi == kEpiFinal || kEpi == kEpiFoldFinal;
    size_t row = static_cast<size_t>(q_row0) + t * kBlockM + (warp & 3) * 32 + lane;   // my query row in the [BH*Nq] views
    if (kEpi == kEpiPartial) row += static_cast<size_t>(blockIdx.z) * gridDim.y * Nq;    // this split's partials
    float lse_prev = 0.f;          // lse_acc[row], the running LSE this pass is folded with (kFold)
    float m_raw = -CUDART_INF_F;   // running (lazy) row max of the unscaled scores
    float m_sc = -CUDART_INF_F;    // m_raw * scale_log2
    float l = 0.f;                 // running row sum of exp2(s*scale_log2 - m_sc)
    const float2 sc2 = make_float2(scale_log2, scale_log2);
    if constexpr (Cfg::kColSplit) {
      // ---- column-split main loop: this thread owns keys [64 hh, 64 hh + 64) of its query row
      const int row_t = (warp & 3) * 32 + lane;
      float* xch_t = xch + t * (2 * 2 * 128);                  // [parity][half][row]
      // the two warps that share 32 query rows (one per half) meet on their own named barrier: the rescale decision
      // below is taken per warp, so nothing wider may be waited for
      const int pair_bar = 1 + t * 4 + (warp & 3);
      for (int j = 0; j < n_kv; ++j) {
        const int n = 2 * j + t, buf = Cfg::kSBufs == 2 ? t : n % Cfg::kSBufs;
        const uint32_t tSb = tmem + buf * kBlockN + lane_off;
        mbar_wait(&s_full[buf], (Cfg::kSBufs == 2 ? j : n / Cfg::kSBufs) & 1);
        tc_fence_after();
        uint32_t s[64];
        auto piece = [&](int c) -> uint32_t(&)[32] { return *reinterpret_cast<uint32_t(*)[32]>(&s[c * 32]); };
        auto piece_max = [&](int c, float& a, float& b) {
#pragma unroll
          for (int i = 0; i < 32; i += 4) {
            a = fmax3(a, __uint_as_float(s[c * 32 + i]), __uint_as_float(s[c * 32 + i + 1]));
            b = fmax3(b, __uint_as_float(s[c * 32 + i + 2]), __uint_as_float(s[c * 32 + i + 3]));
          }
        };
        float mx0 = -CUDART_INF_F, mx1 = -CUDART_INF_F;
        tmem_ld_x32(tSb + hh * 64, piece(0));
        tmem_ld_x32(tSb + hh * 64 + 32, piece(1));
        tmem_wait_ld_x32(piece(0));
        piece_max(0, mx0, mx1);
        tmem_wait_ld_x32(piece(1));
        piece_max(1, mx0, mx1);
        // exchange the half-row maxima; the barrier also tells each half that the other has its scores in registers,
        // so P (which overwrites the first 64 columns of the score buffer) may be written
        float* slot = xch_t + (j & 1) * 256;
        slot[hh * 128 + row_t] = fmaxf(mx0, mx1);
        named_bar_sync(pair_bar, 64);
        const float mx = fmaxf(fmaxf(mx0, mx1), slot[(hh ^ 1) * 128 + row_t]);
        const bool grow = (mx - m_raw) * scale_log2 > kRescaleThreshold;
        if (__any_sync(0xffffffffu, grow)) {                   // same rows, same maxima: both halves decide alike
          const float m_new = fmaxf(m_raw, mx);
          const float alpha = ex2((m_raw - m_new) * scale_log2);
          l *= alpha;
          if (j > 0) {
            if (Cfg::kSBufs > 2) {
              mbar_wait(&pv_done[t], (j - 1) & 1);
              tc_fence_after();
            }
            uint32_t o[kD / 2];                                // my half of the O columns
#pragma unroll
            for (int c = 0; c < kD / 64; ++c) tmem_ld_x32(tO + hh * (kD / 2) + c * 32, *reinterpret_cast<uint32_t(*)[32]>(&o[c * 32]));
            tmem_wait_ld();
#pragma unroll
            for (int i = 0; i < kD / 2; ++i) o[i] = __float_as_uint(__uint_as_float(o[i]) * alpha);
#pragma unroll
            for (int c = 0; c < kD / 64; ++c) tmem_st_x32(tO + hh * (kD / 2) + c * 32, *reinterpret_cast<uint32_t(*)[32]>(&o[c * 32]));
            tmem_wait_st();
            tc_fence_before();
            named_bar_sync(pair_bar, 64);                      // these rows of O_t are rescaled in full before either half releases P
            tc_fence_after();
          }
          m_raw = m_new;
          m_sc = m_new * scale_log2;
        }
        const float2 nm2 = make_float2(-m_sc, -m_sc);
        float2 la = make_float2(0.f, 0.f), lb = make_float2(0.f, 0.f);
#pragma unroll
        for (int c = 0; c < 2; ++c) {
          uint32_t pk[16];
#pragma unroll
          for (int i = 0; i < 32; i += 4) {
            const float2 x0 = ffma2(make_float2(__uint_as_float(s[c * 32 + i]), __uint_as_float(s[c * 32 + i + 1])), sc2, nm2);
            const float2 x1 = ffma2(make_float2(__uint_as_float(s[c * 32 + i + 2]), __uint_as_float(s[c * 32 + i + 3])), sc2, nm2);
            const float2 p0 = ((Cfg::kPolyMask >> (i / 2)) & 1) ? ex2_poly2<RINGX_FWD_POLY_DEGREE>(x0)
                                                                : make_float2(ex2(x0.x), ex2(x0.y));
            const float2 p1 = ((Cfg::kPolyMask >> (i / 2 + 1)) & 1) ? ex2_poly2<RINGX_FWD_POLY_DEGREE>(x1)
                                                                    : make_float2(ex2(x1.x), ex2(x1.y));
            la = fadd2(la, p0);
            lb = fadd2(lb, p1);
            pk[i / 2] = pack_bf16x2(p0.x, p0.y);
            pk[i / 2 + 1] = pack_bf16x2(p1.x, p1.y);
          }
          tmem_st_x16(tSb + hh * 32 + c * 16, pk);
        }
        tmem_wait_st();
        tc_fence_before();
        if (Cfg::kSBufs > 2 && j > 0) mbar_wait(&pv_done[t], (j - 1) & 1);   // (see the unsplit loop)
        mbar_arrive(&p_full[2 * t + hh]);
        l += (la.x + la.y) + (lb.x + lb.y);
      }
      // the row sum over all 128 keys of every tile = the two halves' sums (same reference max)
      mbar_wait(&o_full[t], 0);                                // (also: every named barrier of the loop is behind us)
      float* slot = xch_t + (n_kv & 1) * 256;
      slot[hh * 128 + row_t] = l;
      // Both halves of a row read the running lse, and half 0 overwrites it when the fold is in place (lse_out == lse_acc):
      // the read sits BEFORE the pair barrier, the write after it, so the partner's read cannot see the merged value.
      if (kFold) lse_prev = lse_acc[row];
      named_bar_sync(pair_bar, 64);
      l += slot[(hh ^ 1) * 128 + row_t];
    } else {
      for (int j = 0; j < n_kv; ++j) {
        const int n = 2 * j + t, buf = Cfg::kSBufs == 2 ? t : n % Cfg::kSBufs;     // this tile's scores are S number n
        const uint32_t tS = tmem + buf * kBlockN + lane_off;
        mbar_wait(&s_full[buf], (Cfg::kSBufs == 2 ? j : n / Cfg::kSBufs) & 1);
        tc_fence_after();
        // ---- pass 1: stream S_t(j) out of TMEM; the row max of piece c is taken while piece c+1 is in flight
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
        const float mx = fmaxf(fmaxf(mx0, mx1), fmaxf(mx2, mx3));
        const bool grow = (mx - m_raw) * scale_log2 > kRescaleThreshold;
        if (__any_sync(0xffffffffu, grow)) {
          const float m_new = fmaxf(m_raw, mx);
          const float alpha = ex2((m_raw - m_new) * scale_log2);   // 0 on the first tile (m_raw = -inf)
          l *= alpha;
          if (j > 0) {
            if (Cfg::kSBufs > 2) {     // the scores ran ahead of O_t += P_t(j-1) V: wait for it before touching O_t
              mbar_wait(&pv_done[t], (j - 1) & 1);
              tc_fence_after();
            }
#pragma unroll
            for (int c = 0; c < kD / 32; ++c) {
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
        // ---- pass 2: P = exp2(s * scale_log2 - m_sc), bf16, into the first 64 columns of S_t; row sum in fp32
        const float2 nm2 = make_float2(-m_sc, -m_sc);
        float2 la = make_float2(0.f, 0.f), lb = make_float2(0.f, 0.f);
#pragma unroll
        for (int c = 0; c < kBlockN / 32; ++c) {
          uint32_t pk[16];
#pragma unroll
          for (int i = 0; i < 32; i += 4) {
            const float2 x0 = ffma2(make_float2(__uint_as_float(s[c * 32 + i]), __uint_as_float(s[c * 32 + i + 1])), sc2, nm2);
            const float2 x1 = ffma2(make_float2(__uint_as_float(s[c * 32 + i + 2]), __uint_as_float(s[c * 32 + i + 3])), sc2, nm2);
            const float2 p0 = ((Cfg::kPolyMask >> (i / 2)) & 1) ? ex2_poly2<RINGX_FWD_POLY_DEGREE>(x0)
                                                                : make_float2(ex2(x0.x), ex2(x0.y));
            const float2 p1 = ((Cfg::kPolyMask >> (i / 2 + 1)) & 1) ? ex2_poly2<RINGX_FWD_POLY_DEGREE>(x1)
                                                                    : make_float2(ex2(x1.x), ex2(x1.y));
            la = fadd2(la, p0);
            lb = fadd2(lb, p1);
            pk[i / 2] = pack_bf16x2(p0.x, p0.y);
            pk[i / 2 + 1] = pack_bf16x2(p1.x, p1.y);
          }
          tmem_st_x16(tS + c * 16, pk);
          if (c & 1) {                       // 64 keys of P are in TMEM: let the tensor core start on them
            tmem_wait_st();
            tc_fence_before();
            // (with the scores running ahead, P_t(j) could otherwise complete p_full a second time before the MMA warp
            // has seen P_t(j-1): PV_t(j-1) complete proves it has)
            if (Cfg::kSBufs > 2 && c == 1 && j > 0) mbar_wait(&pv_done[t], (j - 1) & 1);
            mbar_arrive(&p_full[2 * t + (c >> 1)]);
          }
        }
        l += (la.x + la.y) + (lb.x + lb.y);
      }
    }
    // ---- chunk epilogue: loc_out = O / l, loc_lse = m*scale + ln l  (natural log of the scaled scores)
    mbar_wait(&o_full[t], 0);
    tc_fence_after();
    float lse_row = (m_sc + lg2(l)) * 0.6931471805599453f;
    float cb = 1.0f / l, ca = 0.f;            // out = ca * o_acc + cb * O  (O = unnormalised accumulator in TMEM)
    if (kFold) {                              // Eq. 5, two operands: (o_acc, lse_acc) and (loc_out, loc_lse)
      const float la = Cfg::kColSplit ? lse_prev : lse_acc[row];
      const float m = fmaxf(la, lse_row);
      const float wa = ex2((la - m) * 1.4426950408889634f), wb = ex2((lse_row - m) * 1.4426950408889634f);
      const float den = wa + wb, r = 1.0f / den;
      ca = wa * r;
      cb *= wb * r;
      lse_row = m + lg2(den) * 0.6931471805599453f;
    }
#pragma unroll
    for (int c = 0; c < kD / 32; ++c) {
      if (Cfg::kColSplit && c / (kD / 64) != hh) continue;     // column split: each half stores its half of the row
      uint32_t o[32];
      tmem_ld_x32(tO + c * 32, o);
      float4 acc[8];
      if (kFold) {
        const float4* src = reinterpret_cast<const float4*>(o_acc + row * kD + c * 32);
#pragma unroll
        for (int i = 0; i < 8; ++i) acc[i] = __ldcs(src + i);
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
      if (kOutBf16) {
        uint4* dst = reinterpret_cast<uint4*>(static_cast<__nv_bfloat16*>(o_out) + row * kD + c * 32);
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
        float4* dst = reinterpret_cast<float4*>(static_cast<float*>(o_out) + row * kD + c * 32);
#pragma unroll
        for (int i = 0; i < 8; ++i) dst[i] = make_float4(r[i * 4], r[i * 4 + 1], r[i * 4 + 2], r[i * 4 + 3]);
      }
    }
    if (hh == 0) lse_out[row] = lse_row;
  } else {
    setmaxnreg_dec<Cfg::kAuxRegs>();   // the two idle warps of the last warpgroup: release their registers
  }

  tc_fence_before();
  __syncthreads();
  if (warp == Cfg::kProducerWarp) tmem_dealloc<512>(tmem);
}

template <int kD, int kEpi>
cudaError_t launch_t(const CUtensorMap& mq, const CUtensorMap& mk, const CUtensorMap& mv, void* o_out, float* lse_out,
                     const float* o_acc, const float* lse_acc, int BH, int Nq, int nk_stride, int k_off, int nk,
                     float scale, int splits, cudaStream_t stream) {
  using Cfg = FwdCfg<kD>;
  auto kern = attn_chunk_fwd_kernel<kD, kEpi>;
  static unsigned char configured[kMaxDevices];
  if (cudaError_t e = set_max_dyn_smem_once(kern, Cfg::kSmemBytes, configured); e != cudaSuccess) return e;
  dim3 grid(Nq / (2 * kBlockM), BH, splits);
  kern<<<grid, Cfg::kThreads, Cfg::kSmemBytes, stream>>>(mq, mk, mv, o_out, lse_out, o_acc, lse_acc, Nq, nk_stride, k_off,
                                                       nk / kBlockN / splits, scale * 1.4426950408889634f);
  count_launch();
  return cudaGetLastError();
}

template <int kD>
cudaError_t launch_d(int epi, const CUtensorMap& mq, const CUtensorMap& mk, const CUtensorMap& mv, void* o_out,
                     float* lse_out, const float* o_acc, const float* lse_acc, int BH, int Nq, int nk_stride, int k_off,
                     int nk, float scale, int splits, cudaStream_t stream) {
  switch (epi) {
    case kEpiPartial:
      return launch_t<kD, kEpiPartial>(mq, mk, mv, o_out, lse_out, o_acc, lse_acc, BH, Nq, nk_stride, k_off, nk, scale, splits, stream);
    case kEpiFinal:
      return launch_t<kD, kEpiFinal>(mq, mk, mv, o_out, lse_out, o_acc, lse_acc, BH, Nq, nk_stride, k_off, nk, scale, splits, stream);
    case kEpiFold:
      return launch_t<kD, kEpiFold>(mq, mk, mv, o_out, lse_out, o_acc, lse_acc, BH, Nq, nk_stride, k_off, nk, scale, splits, stream);
    default:
      return launch_t<kD, kEpiFoldFinal>(mq, mk, mv, o_out, lse_out, o_acc, lse_acc, BH, Nq, nk_stride, k_off, nk, scale, splits, stream);
  }
}

}  // namespace

cudaError_t launch_attn_chunk_fwd_sm100(const void* q, const void* k, const void* v, void* o_out, float* lse_out,
                                        const float* o_acc, const float* lse_acc, int BH, int Nq, int nk_stride,
                                        int k_off, int nk, int d, float scale, int epilogue, int splits,
                                        cudaStream_t stream) {
  if (splits < 1 || (splits > 1 && epilogue != kFwdEpiPartial) || (nk / 128) % splits) return cudaErrorInvalidValue;
  CUtensorMap mq, mk, mv;
  const CUtensorMapDataType dt = CU_TENSOR_MAP_DATA_TYPE_BFLOAT16;
  if (!make_tmap_2d(&mq, q, dt, 2, (uint64_t)BH * Nq, d, 128, 64, kSwizzle128B) ||
      !make_tmap_2d(&mk, k, dt, 2, (uint64_t)BH * nk_stride, d, 128, 64, kSwizzle128B) ||
      !make_tmap_2d(&mv, v, dt, 2, (uint64_t)BH * nk_stride, d, 128, 64, kSwizzle128B))
    return cudaErrorInvalidValue;
  if (d == 64) return launch_d<64>(epilogue, mq, mk, mv, o_out, lse_out, o_acc, lse_acc, BH, Nq, nk_stride, k_off, nk, scale, splits, stream);
  return launch_d<128>(epilogue, mq, mk, mv, o_out, lse_out, o_acc, lse_acc, BH, Nq, nk_stride, k_off, nk, scale, splits, stream);
}

}  // namespace ringx

