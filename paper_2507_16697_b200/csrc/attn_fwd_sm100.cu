// attn_fwd_sm100.cu -- one KV-chunk pass of the forward on tcgen05 tensor cores.
//
// For every query row of a [128 x 2]-row work item and the keys [k_off, k_off + nk) of its head:
//   loc_out = softmax(scale q K_c^T) V_c,  loc_lse = log sum_j exp(scale q.k_j)      (Eq. 1/3/4)
// bf16 operands, fp32 accumulation ("mixed float32-bfloat16").
// Any sequence length: Q, K, V are addressed through [BH][rows][d] tensor maps, so rows and keys past the end of a head
// read as zeros; such rows are computed like any other and never stored, such keys get a score of -inf (kTail).
//
// PERSISTENT kernel with hardware work stealing (cluster launch control).  The grid is one CTA per work item (item =
// 256 query rows of one head [x one key split]; blockIdx.x = query tile, so the CTAs running at any time share one
// head's K,V chunk in L2), but a CTA that has finished its item does not exit: it asks the block scheduler to CANCEL
// the launch of a CTA that has not started yet (clusterlaunchcontrol.try_cancel) and takes over its block index, until
// none is left.  So only one wave of CTAs ever starts; TMEM is allocated and the mbarriers are initialised once per
// SM; items are handed out dynamically in launch order; and the tensor-core stream does not stop at an item boundary: score MMAs of item n+1 are issued behind the
// last P V MMAs of item n ("seamless"), the softmax warps go from the epilogue of item n straight to scores that are
// already waiting.  Measured against one CTA per item: C2 forward (32 key tiles per item) 759 -> 785 TFLOP/s, C4 817 -> 822,
// C3 (256 tiles per item) unchanged.  If the hardware grants no cancellation the kernel is simply the
// one-item-per-CTA kernel: correctness never depends on a request succeeding.
//
// Roles (d = 128: 384 threads, d = 64: 640 threads; registers re-split with setmaxnreg):
//   softmax warpgroups   d = 128: warps 0-3 / 4-7 = query tile 0 / 1 (thread = one query row = one TMEM lane)
//                        d = 64 : warps 0-3, 4-7 = the two 64-key halves of every score tile of query tile 0,
//                                 warps 8-11, 12-15 = the same for query tile 1 (column split, see FwdCfg)
//   K/V producer warp    the TMA ring of K and V tiles, in the order the MMA warp consumes them, across items
//   MMA warp             one elected lane: S_t = Q_t K_j^T (SS), O_t += P_t V_j (P from TMEM, V MN-major)
//   aux producer warp    the work-item scheduler (one cancellation request ahead; responses go round a 2-slot ring in
//                        shared memory that every other warp reads), and per item: the Q tiles (as soon as the last
//                        score MMA of the previous item has read them), an L2 prefetch of the next item's Q, and
//                        -- d = 64, fold epilogues -- the item's fp32 o_acc tile
//   (one more warp idles: it completes the last warpgroup so that setmaxnreg can be used)
// TMEM columns (d = 128): S_0 [0,128) S_1 [128,256) O_0 [256,384) O_1 [384,512); P_t (bf16) overwrites the first 64
// columns of S_t.  The two query tiles ping-pong: while warpgroup t turns S_t into P_t the tensor core works on tile
// 1-t.  The MMA pipe executes in issue order, so S_t(j+1) -- issued right after O_t += P_t(j) V_j -- cannot overwrite
// P_t(j) early, and the commit that signals S_t(j+1) also proves O_t(j) complete: the softmax warps may rescale O_t in
// place without a further barrier.
// d = 64 has 128 TMEM columns to spare and uses them for a third score buffer: S number g (counted over the whole
// stream of the CTA; g even = tile 0) goes to buffer g % 3 [0,384), O_0 [384,448), O_1 [448,512), and is issued behind
// PV number g - 3, i.e. one tile ahead, so a softmax warpgroup finds its next scores waiting (ring order K K V K V ...).
// Running ahead of PV_t(j-1) costs two waits on pv_done[t]: before the (rare) in-place rescale of O_t, and before
// P_t(j) is signalled (so that p_full cannot complete twice before the MMA warp has seen it once).
// Online softmax in the exp2 domain with a lazy running max (O, l are only rescaled when the row max grew by more than
// 2^8), so the rescale is off the common path.  The softmax streams S out of TMEM in 32-column pieces (the row max of
// piece c is taken while piece c+1 is in flight), uses the packed FFMA2/FADD2 and three-input FMNMX3 forms, and hands
// P to the tensor core in two 64-key halves so that the first half of O += P V starts while the second half of P is
// still being exponentiated.
#include <type_traits>

#include "kernels.cuh"

namespace ringx {
namespace {

using namespace ptx;

constexpr int kBlockM = 128;          // query rows per tile (= TMEM lanes)
constexpr int kBlockN = 128;          // keys per KV tile
constexpr float kRescaleThreshold = 8.0f;   // log2 units
// d = 64 is bound by the softmax warps (one exponential per 4*64 tensor FLOPs: 2048 clk of MUFU.EX2 against 1024 clk
// of MMA per 128-key iteration; ncu r02a: XU pipe 72 % busy, tensor pipe 41 %).  Of the 16 element pairs of every
// 32-key piece, those in this mask take 2^x from the FMA-pipe polynomial ptx::ex2_poly2 (degree 4, relative error
// 2.7e-6: P also feeds the fp32 row sum behind LSE).  Measured on C4 forward: 0 -> 781, 1/8 -> 796, 1/4 -> 791 TFLOP/s
// (the warps are close to issue-bound as well).  d = 128 is balanced and power-capped: it stays on the MUFU.
constexpr unsigned kPolyMaskD64 = 0x8080;
constexpr int kPolyDegree = 4;

template <int kD>
struct FwdCfg {
  static constexpr int kPanels = kD / 64;                    // 64 bf16 = one 128-byte swizzle row
  static constexpr int kPanelBytes = 128 * 128;              // 128 rows x 128 B
  static constexpr int kTileBytes = kPanels * kPanelBytes;   // Q, K or V tile
  static constexpr unsigned kPolyMask = kD == 64 ? kPolyMaskD64 : 0u;
  // Score buffers in TMEM.  d = 128: one per query tile (2 x 128 + 2 x 128 O columns = 512).  d = 64 leaves 128
  // columns, enough for a third buffer: the score MMAs then run one tile ahead.
  static constexpr int kSBufs = kD == 128 ? 2 : 3;
  static constexpr int kKLead = (kSBufs + 1) / 2;            // K tiles the ring holds ahead of the V tile of the same index
  static constexpr uint32_t kOBase = kSBufs * 128;           // O_t at kOBase + t * kD
  static constexpr int kBarBytes = 512;
  // Column split (d = 64): the 128 keys of a score tile are shared by TWO softmax warpgroups (64 keys each), i.e. four
  // softmax warpgroups per CTA and four warps per scheduler instead of two -- the MUFU pipe then stays busy while
  // other warps are in their TMEM-load / row-max phase or wait on a barrier.  The two halves of a row exchange their
  // row maxima (and, in the epilogue, their row sums) through shared memory.  (At d = 128 the same split ran at 587
  // against 1270 TFLOP/s: not used there.)
  static constexpr bool kColSplit = kD == 64;
  // Fold epilogues at d = 64 read the item's running fp32 o_acc tile [256, 64] from shared memory, where the aux warp
  // put it by TMA during the item: the epilogue then costs the softmax warps a few hundred clocks instead of a global
  // round trip.  (d = 128 has no shared memory to spare and 8 x longer items: it reads o_acc from global memory.)
  static constexpr bool kOaccSmem = kD == 64;
  static constexpr int kOaccBytes = kOaccSmem ? 4 * kPanelBytes : 0;      // 4 panels of [128 rows][32 fp32], 128B-swizzled
  static constexpr int kStages = kD == 128 ? 5 : 7;          // K/V ring slots
  static constexpr int kSoftmaxWarps = kColSplit ? 16 : 8;
  static constexpr int kProducerWarp = kSoftmaxWarps, kMmaWarp = kSoftmaxWarps + 1, kAuxWarp = kSoftmaxWarps + 2;
  static constexpr int kThreads = (kSoftmaxWarps + 4) * 32;
  // setmaxnreg moves registers inside the CTA's own pool (threads x the launch-time count: 384 x 168 / 640 x 96), so what
  // the softmax warpgroups gain must equal what the last warpgroup gives up: 256 x (224-168) = 128 x (168-56);
  // 512 x (112-96) = 128 x (96-32)
  static constexpr int kSoftmaxRegs = kColSplit ? 112 : 224;
  static constexpr int kAuxRegs = kColSplit ? 32 : 56;
  static constexpr int kXchBytes = kColSplit ? 2 * 3 * 2 * 128 * 4 : 0;    // [tile][slot][half][row] floats
  static constexpr int kSmemBytes = 1024 + 2 * kTileBytes + kStages * kTileBytes + kOaccBytes + kBarBytes + kXchBytes;
};

// Epilogue modes (kEpi): what happens to (loc_out, loc_lse) of this chunk
//   kEpiPartial   written as they are, fp32                       (first pass; ringx_attn_chunk_fwd)
//   kEpiFinal     loc_out written as bf16                         (single pass: the chunk is the whole sequence)
//   kEpiFold      folded into the running (o_acc, lse_acc) with the two-operand Eq. 5, in place, fp32
//   kEpiFoldFinal folded with (o_acc, lse_acc) and written to (o_out, lse_out) as bf16 (last pass)
// Folding here instead of in a separate lse_merge launch saves the round trip of loc_out through HBM; it is the same
// arithmetic as merge.cu's lse_merge_kernel, row by row (a thread owns a query row).
enum { kEpiPartial = 0, kEpiFinal = 1, kEpiFold = 2, kEpiFoldFinal = 3 };

struct FwdParams {
  void* o_out;
  float* lse_out;
  const float* o_acc;
  const float* lse_acc;
  int Nq, nk_stride, k_off, n_kv;      // n_kv = key tiles per item
  int k_tail;                          // keys of the pass's last key tile that exist (0: all 128) -- a ragged sequence
  float scale_log2;
};

// A work item = a block index of the launch grid: (query tile, head, key split).
struct ItemId {
  int qt, bh, z;
  bool valid;
};
struct ItemRows {
  int bh;            // head: the third TMA coordinate of the [BH][rows][d] views
  int q_in;          // first query row of the item within its head (rows >= Nq do not exist: loaded as zero, never stored)
  int k_in;          // first key row within the head
  int q_row0;        // first query row in the flat [BH*Nq, d] view (global-memory addressing of o_acc, lse_acc)
  size_t out_row0;   // first row of (o_out, lse_out): q_row0, plus the split's offset for partials
};
template <int kEpi>
__device__ __forceinline__ ItemRows item_rows(const FwdParams& p, const ItemId& id) {
  ItemRows r;
  r.bh = id.bh;
  r.q_in = id.qt * (2 * kBlockM);
  r.k_in = p.k_off + id.z * p.n_kv * kBlockN;                             // z = key split (split-KV; partials only)
  r.q_row0 = id.bh * p.Nq + r.q_in;
  r.out_row0 = static_cast<size_t>(r.q_row0) + (kEpi == kEpiPartial ? static_cast<size_t>(id.z) * gridDim.y * p.Nq : 0);
  return r;
}

// kTail: the pass ends in a key tile with fewer than 128 keys (a ragged sequence; prm.k_tail of them exist).  A separate
// instantiation, so that the mask costs the full-tile kernels neither an instruction nor a register (the d = 64 softmax
// warps have none to spare: with the mask compiled in they spill inside the loop, -2 % on C2 / C4).
template <int kD, int kEpi, bool kTail>
__global__ void __launch_bounds__(FwdCfg<kD>::kThreads, 1)
attn_chunk_fwd_kernel(const __grid_constant__ CUtensorMap map_q, const __grid_constant__ CUtensorMap map_k,
                      const __grid_constant__ CUtensorMap map_v, const __grid_constant__ CUtensorMap map_oacc,
                      const FwdParams prm) {
  using Cfg = FwdCfg<kD>;
  constexpr bool kFold = kEpi == kEpiFold || kEpi == kEpiFoldFinal;
  constexpr bool kOutBf16 = kEpi == kEpiFinal || kEpi == kEpiFoldFinal;
  constexpr bool kOaccSmem = kFold && Cfg::kOaccSmem;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t* sQ = smem;
  uint8_t* sKV = smem + 2 * Cfg::kTileBytes;
  uint8_t* sOacc = sKV + Cfg::kStages * Cfg::kTileBytes;
  uint64_t* bars = reinterpret_cast<uint64_t*>(sOacc + Cfg::kOaccBytes);
  uint64_t* q_full = bars;                  // [2]  aux -> MMA: Q_t of the item in shared memory
  uint64_t* q_empty = bars + 2;             // [2]  MMA -> aux: the last score MMA of the item has read Q_t
  uint64_t* s_full = bars + 4;              // [kSBufs] MMA -> softmax: score buffer b holds S number g (g % kSBufs == b)
  uint64_t* p_full = bars + 7;              // [2][2] softmax -> MMA: half h (64 keys) of P_t(j) in TMEM (O_t rescaled if needed)
  uint64_t* o_full = bars + 11;             // [2]  MMA -> softmax: last O_t of the item complete
  uint64_t* pv_done = bars + 13;            // [2]  MMA -> softmax: O_t += P_t(j) V_j complete (used when kSBufs > 2)
  uint64_t* oacc_full = bars + 15;          // aux -> softmax: the item's o_acc tile in shared memory
  uint64_t* oacc_empty = bars + 16;         // softmax -> aux: every thread has read its part of it
  uint64_t* kv_full = bars + 17;            // [kStages]
  uint64_t* kv_empty = bars + 17 + Cfg::kStages;
  uint64_t* sched_full = bars + 17 + 2 * Cfg::kStages;      // [2] scheduler -> all: response of request r in slot r & 1
  uint64_t* sched_empty = sched_full + 2;                   // [2] all -> scheduler: every consumer warp has read it
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(sched_empty + 2);
  uint8_t* sched_resp = reinterpret_cast<uint8_t*>(bars) + 384;      // 2 x 16 bytes
  float* xch = reinterpret_cast<float*>(reinterpret_cast<uint8_t*>(bars) + Cfg::kBarBytes);   // column-split exchange

  const int warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0);   // provably warp-uniform: keeps MMA/TMA operands in uniform registers
  const int lane = threadIdx.x & 31;
  const int n_kv = prm.n_kv;
  // Work items after the CTA's own block come from the scheduler's ring: request r (r = 0, 1, ...) yields local item
  // r + 1, or "none left".  Every consumer WARP calls this exactly once per request, all lanes together.
  auto next_item = [&](int r) -> ItemId {
    const int s = r & 1;
    mbar_wait(&sched_full[s], (r >> 1) & 1);
    ItemId id;
    id.valid = clc_query(sched_resp + 16 * s, id.qt, id.bh, id.z);
    __syncwarp();
    if (lane == 0) mbar_arrive(&sched_empty[s]);
    return id;
  };
  ItemId own;
  own.qt = blockIdx.x; own.bh = blockIdx.y; own.z = blockIdx.z; own.valid = true;

  if (threadIdx.x == 0) {
    for (int i = 0; i < 2; ++i) {
      mbar_init(&q_full[i], 1);
      mbar_init(&q_empty[i], 1);
      mbar_init(&p_full[2 * i], kBlockM);
      mbar_init(&p_full[2 * i + 1], kBlockM);
      mbar_init(&o_full[i], 1);
      mbar_init(&pv_done[i], 1);
    }
    for (int i = 0; i < Cfg::kSBufs; ++i) mbar_init(&s_full[i], 1);
    mbar_init(oacc_full, 1);
    mbar_init(oacc_empty, Cfg::kSoftmaxWarps * 32);
    for (int i = 0; i < 2; ++i) {
      mbar_init(&sched_full[i], 1);
      mbar_init(&sched_empty[i], Cfg::kSoftmaxWarps + 2);    // softmax warps + K/V producer + MMA warp
    }
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
      if (kOaccSmem) prefetch_tmap(&map_oacc);
    }
    tmem_alloc<512>(tmem_slot);
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_slot;

  if (warp == Cfg::kProducerWarp) {
    setmaxnreg_dec<Cfg::kAuxRegs>();
    // ------------------------------------------------------------------ K/V producer
    // (the whole warp runs the loop so that every operand is warp-uniform; one elected lane issues)
    // Ring order = the order in which the MMA warp first touches the tiles.  With the key tiles of all this CTA's
    // items numbered g = 0, 1, ... in one stream:  K_0 .. K_{kKLead-1}, then V_g, K_{g+kKLead} for g = 0, 1, ...
    //   kSBufs = 2: K_0 V_0 K_1 V_1 ...        kSBufs = 3: K_0 K_1 V_0 K_2 V_1 K_3 ...
    const bool leader = elect_one();
    const uint64_t pol_kv = policy_evict_last();
    // The K cursor runs kKLead tiles ahead of the V cursor, possibly into later items: it is the one that asks the
    // scheduler for items; their first key rows wait in a 3-deep register FIFO for the V cursor.
    int stage = 0, phase = 0;
    auto push = [&](const CUtensorMap* map, int row, int head) {
      mbar_wait_relaxed(&kv_empty[stage], phase ^ 1);
      if (leader) {
        uint8_t* dst = sKV + stage * Cfg::kTileBytes;
        mbar_arrive_expect_tx(&kv_full[stage], Cfg::kTileBytes);
#pragma unroll
        for (int p = 0; p < Cfg::kPanels; ++p)
          tma_load_3d(dst + p * Cfg::kPanelBytes, map, &kv_full[stage], p * 64, row, head, pol_kv);
      }
      __syncwarp();
      if (++stage == Cfg::kStages) { stage = 0; phase ^= 1; }
    };
    // FIFO of (first key row in the head, head): f0 = the V cursor's item
    int f0 = item_rows<kEpi>(prm, own).k_in, f1 = 0, f2 = 0, h0 = own.bh, h1 = 0, h2 = 0, fn = 1;
    int k_row = f0, k_head = h0, kj = 0, vj = 0, req = 0;
    bool k_more = true;                     // the K cursor stands in a valid item
    auto push_k = [&]() {
      push(&map_k, k_row + kj * kBlockN, k_head);
      if (++kj == n_kv) {
        kj = 0;
        const ItemId id = next_item(req++);
        k_more = id.valid;
        if (k_more) {
          k_row = item_rows<kEpi>(prm, id).k_in;
          k_head = id.bh;
          if (fn == 1) { f1 = k_row; h1 = k_head; } else { f2 = k_row; h2 = k_head; }   // (fn <= 2 here: at most 2 items ahead)
          ++fn;
        }
      }
    };
    for (int i = 0; i < Cfg::kKLead && k_more; ++i) push_k();
    while (fn > 0) {
      push(&map_v, f0 + vj * kBlockN, h0);
      if (++vj == n_kv) { vj = 0; f0 = f1; f1 = f2; h0 = h1; h1 = h2; --fn; }
      if (k_more) push_k();
    }
  } else if (warp == Cfg::kAuxWarp) {
    setmaxnreg_dec<Cfg::kAuxRegs>();
    // ------------------------------------------------------------------ aux producer: Q tiles and the o_acc tile of every item
    const bool leader = elect_one();
    const uint64_t pol_q = policy_evict_first();
    ItemId cur = own;
    for (int li = 0;; ++li) {
      const ItemRows it = item_rows<kEpi>(prm, cur);
      // ---- request the next item (request number li) while this one runs
      const int sl = li & 1;
      if (li >= 2) mbar_wait_relaxed(&sched_empty[sl], ((li >> 1) & 1) ^ 1);   // request li-2 has been read by every warp
      fence_proxy_async_smem();                                               // (their generic reads before the async write)
      if (leader) {
        mbar_arrive_expect_tx(&sched_full[sl], 16);
        clc_try_cancel(sched_resp + 16 * sl, &sched_full[sl]);
      }
      __syncwarp();
      // ---- this item's Q tiles
#pragma unroll
      for (int t = 0; t < 2; ++t) {
        if (li > 0) mbar_wait_relaxed(&q_empty[t], (li - 1) & 1);      // the previous item's score MMAs are done with Q_t
        if (leader) {
          mbar_arrive_expect_tx(&q_full[t], Cfg::kTileBytes);
#pragma unroll
          for (int p = 0; p < Cfg::kPanels; ++p)
            tma_load_3d(sQ + t * Cfg::kTileBytes + p * Cfg::kPanelBytes, &map_q, &q_full[t], p * 64,
                        it.q_in + t * kBlockM, it.bh, pol_q);
        }
        __syncwarp();
      }
      if (kOaccSmem) {
        if (li > 0) mbar_wait_relaxed(oacc_empty, (li - 1) & 1);       // the previous epilogue has read its tile
        if (leader) {
          mbar_arrive_expect_tx(oacc_full, Cfg::kOaccBytes);
#pragma unroll
          for (int p = 0; p < 4; ++p)           // panel p = (query tile p >> 1, columns [32 (p & 1), +32))
            tma_load_3d(sOacc + p * Cfg::kPanelBytes, &map_oacc, oacc_full, (p & 1) * 32, it.q_in + (p >> 1) * kBlockM,
                        it.bh, pol_q);
        }
        __syncwarp();
      }
      // ---- the scheduler's answer: the next item, or none (after which no further request may be made)
      mbar_wait_relaxed(&sched_full[sl], (li >> 1) & 1);
      cur.valid = clc_query(sched_resp + 16 * sl, cur.qt, cur.bh, cur.z);
      if (!cur.valid) break;
      if (leader) {                             // its Q: into L2 now, so that the load at the item boundary is an L2 hit
        const int nq0 = item_rows<kEpi>(prm, cur).q_in;
#pragma unroll
        for (int t = 0; t < 2; ++t)
#pragma unroll
          for (int p = 0; p < Cfg::kPanels; ++p) tma_prefetch_3d(&map_q, p * 64, nq0 + t * kBlockM, cur.bh);
      }
      __syncwarp();
    }
  } else if (warp == Cfg::kMmaWarp) {
    // ------------------------------------------------------------------ MMA issuer
    setmaxnreg_dec<Cfg::kAuxRegs>();
    const bool leader = elect_one();
    constexpr uint32_t idesc_s = make_idesc_bf16(kBlockM, kBlockN, 0, 0);    // Q (K-major) x K^T (K-major)
    constexpr uint32_t idesc_o = make_idesc_bf16(kBlockM, kD, 0, 1);         // P (TMEM) x V (MN-major)
    const uint32_t q_addr = smem_u32(sQ), kv_addr = smem_u32(sKV);
    int stage = 0, phase = 0;
    auto commit = [&](uint64_t* bar) {
      if (leader) mma_commit(bar);
      __syncwarp();
    };
    // ring slots are taken in the producer's order; a K tile serves two score MMAs (tiles 0, 1), a V tile two PV MMAs
    auto acquire = [&]() {
      const int st = stage;
      mbar_wait(&kv_full[stage], phase);
      tc_fence_after();
      if (++stage == Cfg::kStages) { stage = 0; phase ^= 1; }
      return st;
    };
    // The score MMAs and the PV MMAs of all this CTA's items form two streams, numbered g = 0, 1, ...; within an item
    // number m = 2 j + t (key tile j, query tile t).  S number g goes to score buffer g % kSBufs and is issued behind
    // PV number g - kSBufs.
    const int n_s = 2 * n_kv;
    int k_slot = 0, v_slot = 0;
    int s_m = 0, s_li = 0, s_buf = 0;                // next score MMA: number within its item, local item, score buffer
    int p_j = 0, p_li = 0, p_buf = 0;                // next PV MMA pair: key tile, local item, score buffer of tile 0
    int n_known = 1;                                 // items the score stream has been given so far
    bool s_more = true;                              // the score stream stands in a valid item
    uint32_t p_par = 0;                              // parity of the next p_full completions (same for both query tiles)
    // score MMA on query tile T (the stream alternates T = 0, 1, 0, ...: a compile-time constant at every call site)
    auto score = [&](auto t_c) {
      constexpr int T = decltype(t_c)::value;
      if (T == 0) k_slot = acquire();
      if (s_m < 2) {                                 // first score MMA of the item on this query tile: wait for Q_t
        mbar_wait(&q_full[T], s_li & 1);
        tc_fence_after();
      }
      const int buf = Cfg::kSBufs == 2 ? T : s_buf;
      const uint32_t a0 = q_addr + T * Cfg::kTileBytes, b0 = kv_addr + k_slot * Cfg::kTileBytes;
      if (leader) {
#pragma unroll
        for (int k = 0; k < kD / 16; ++k) {
          const uint32_t off = (k >> 2) * Cfg::kPanelBytes + (k & 3) * 32;
          mma_ss(tmem + buf * kBlockN, make_smem_desc_sw128(a0 + off, 16, 1024), make_smem_desc_sw128(b0 + off, 16, 1024),
                 idesc_s, k > 0);
        }
        mma_commit(&s_full[buf]);
      }
      __syncwarp();
      if (T == 1) commit(&kv_empty[k_slot]);
      if (s_m >= n_s - 2) commit(&q_empty[T]);       // last score MMA of the item on Q_t: the aux warp may reload it
      if (Cfg::kSBufs > 2 && ++s_buf == Cfg::kSBufs) s_buf = 0;
      if (++s_m == n_s) {                            // the score stream enters the next item, if the scheduler has one
        s_m = 0;
        s_more = next_item(s_li++).valid;
        if (s_more) ++n_known;
      }
    };
    // O_t (+)= P V: keys [64*half, 64*half + 64) of the PV MMA (P sits in its score buffer)
    auto issue_o = [&](int buf, int t, int st, int half, bool accumulate) {
      const uint32_t b0 = kv_addr + st * Cfg::kTileBytes;
      if (leader) {
#pragma unroll
        for (int k = half * 4; k < half * 4 + 4; ++k)
          mma_ts(tmem + Cfg::kOBase + t * kD, tmem + buf * kBlockN + k * 8,
                 make_smem_desc_sw128(b0 + k * 2048, Cfg::kPanelBytes, 1024), idesc_o, accumulate || k > 0);
      }
      __syncwarp();
    };
    using T0 = std::integral_constant<int, 0>;
    using T1 = std::integral_constant<int, 1>;
    // prologue: the first kSBufs score tiles
    score(T0{});
    if (s_more) score(T1{});
    if (Cfg::kSBufs > 2 && s_more) score(T0{});
    while (p_li < n_known) {                         // one key tile of the PV stream per iteration: tiles t = 0, 1
#pragma unroll
      for (int t = 0; t < 2; ++t) {
        int buf = t;
        if (Cfg::kSBufs > 2) {
          buf = p_buf;
          if (++p_buf == Cfg::kSBufs) p_buf = 0;
        }
        if (t == 0) v_slot = acquire();
        mbar_wait(&p_full[2 * t], p_par);
        tc_fence_after();
        issue_o(buf, t, v_slot, 0, p_j > 0);
        mbar_wait(&p_full[2 * t + 1], p_par);
        tc_fence_after();
        issue_o(buf, t, v_slot, 1, true);
        if (Cfg::kSBufs > 2) commit(&pv_done[t]);
        if (t == 1) commit(&kv_empty[v_slot]);
        if (p_j + 1 == n_kv) commit(&o_full[t]);                               // last PV of the item on tile t
        if (s_more) {                                                          // refill the score buffer this PV freed
          if ((t + Cfg::kSBufs) & 1) score(T1{}); else score(T0{});
        }
      }
      p_par ^= 1;
      if (++p_j == n_kv) { p_j = 0; ++p_li; }
    }
  } else if (warp < Cfg::kSoftmaxWarps) {
    // ------------------------------------------------------------------ softmax warpgroups
    setmaxnreg_inc<Cfg::kSoftmaxRegs>();
    const int t = Cfg::kColSplit ? warp >> 3 : warp >> 2;      // query tile
    const int hh = Cfg::kColSplit ? (warp >> 2) & 1 : 0;       // column split: which 64 keys of every score tile
    const int row_t = (warp & 3) * 32 + lane;                  // my query row within the tile = TMEM lane
    const uint32_t lane_off = static_cast<uint32_t>((warp & 3) * 32) << 16;
    const uint32_t tO = tmem + Cfg::kOBase + t * kD + lane_off;
    const float scale_log2 = prm.scale_log2;
    const float2 sc2 = make_float2(scale_log2, scale_log2);
    float* xch_t = xch + t * (3 * 2 * 128);                    // [slot][half][row]; slot 2 = the row sums of the epilogue
    // the two warps that share 32 query rows (one per half) meet on their own named barrier: the rescale decision
    // below is taken per warp, so nothing wider may be waited for
    const int pair_bar = 1 + t * 4 + (warp & 3);
    // stream state, carried across items: my next score tile is S number g (advances by 2 per tile, items included)
    int g = t;
    int buf3 = t % Cfg::kSBufs;                                 // g % kSBufs
    uint32_t tile_par = 0;                                      // parity of the number of tiles of my query tile done so far

    ItemId cur = own;
    for (int li = 0; cur.valid; ++li) {
      const ItemRows it = item_rows<kEpi>(prm, cur);
      const size_t row = it.out_row0 + t * kBlockM + row_t;     // my row in (o_out, lse_out)
      // ... in (o_acc, lse_acc); -1 for a row past the end of the head (a ragged sequence): such rows were loaded as
      // zeros, are computed like any other and never stored.  (A sentinel instead of a flag: the d = 64 softmax warps
      // have no register to spare.)
      const long long acc_row = it.q_in + t * kBlockM + row_t < prm.Nq ? static_cast<long long>(it.q_row0) + t * kBlockM + row_t : -1;
      auto row_valid = [&]() { return acc_row >= 0; };
      // the keys past the end of the head in the pass's last key tile (zero rows of K: score 0) are masked to -inf
      // (kTail launches have no key splits)
      auto tail_tile = [&](int j) { return kTail && j == n_kv - 1; };
      float lse_prev = 0.f;                                     // lse_acc of my row: the running LSE this pass is folded with
      if (kFold && row_valid()) lse_prev = prm.lse_acc[acc_row];   // (read at the item's start: long since there at its end)
      float m_raw = -CUDART_INF_F;   // running (lazy) row max of the unscaled scores
      float m_sc = -CUDART_INF_F;    // m_raw * scale_log2
      float l = 0.f;                 // running row sum of exp2(s*scale_log2 - m_sc)
      if constexpr (Cfg::kColSplit) {
        // ---- column-split main loop: this thread owns keys [64 hh, 64 hh + 64) of its query row
        for (int j = 0; j < n_kv; ++j) {
          const int buf = Cfg::kSBufs == 2 ? t : buf3;
          const uint32_t tSb = tmem + buf * kBlockN + lane_off;
          mbar_wait(&s_full[buf], (Cfg::kSBufs == 2 ? tile_par : static_cast<uint32_t>(g / Cfg::kSBufs)) & 1);
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
          if (tail_tile(j)) {                                    // warp-uniform, last key tile of a ragged pass only
#pragma unroll
            for (int c = 0; c < 64; ++c)
              if (hh * 64 + c >= prm.k_tail) s[c] = 0xff800000u;   // -inf
            mx0 = mx1 = -CUDART_INF_F;
            piece_max(0, mx0, mx1);
            piece_max(1, mx0, mx1);
          }
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
                mbar_wait(&pv_done[t], tile_par ^ 1);            // O_t += P_t(j-1) V complete
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
              const float2 p0 = ((Cfg::kPolyMask >> (i / 2)) & 1) ? ex2_poly2<kPolyDegree>(x0) : make_float2(ex2(x0.x), ex2(x0.y));
              const float2 p1 = ((Cfg::kPolyMask >> (i / 2 + 1)) & 1) ? ex2_poly2<kPolyDegree>(x1) : make_float2(ex2(x1.x), ex2(x1.y));
              la = fadd2(la, p0);
              lb = fadd2(lb, p1);
              pk[i / 2] = pack_bf16x2(p0.x, p0.y);
              pk[i / 2 + 1] = pack_bf16x2(p1.x, p1.y);
            }
            tmem_st_x16(tSb + hh * 32 + c * 16, pk);
          }
          tmem_wait_st();
          tc_fence_before();
          // (with the scores running ahead, P_t(j) could otherwise complete p_full a second time before the MMA warp
          // has seen P_t(j-1): PV_t(j-1) complete proves it has.  At j = 0 the epilogue's wait on o_full did that.)
          if (Cfg::kSBufs > 2 && j > 0) mbar_wait(&pv_done[t], tile_par ^ 1);
          mbar_arrive(&p_full[2 * t + hh]);
          l += (la.x + la.y) + (lb.x + lb.y);
          g += 2;
          buf3 += 2;
          if (buf3 >= Cfg::kSBufs) buf3 -= Cfg::kSBufs;
          tile_par ^= 1;
        }
        // the row sum over all 128 keys of every tile = the two halves' sums (same reference max)
        mbar_wait(&o_full[t], li & 1);                             // (also: every named barrier of the loop is behind us)
        float* slot = xch_t + 2 * 256;
        slot[hh * 128 + row_t] = l;
        named_bar_sync(pair_bar, 64);
        l += slot[(hh ^ 1) * 128 + row_t];
      } else {
        for (int j = 0; j < n_kv; ++j) {
          const int buf = Cfg::kSBufs == 2 ? t : buf3;               // this tile's scores are S number g
          const uint32_t tS = tmem + buf * kBlockN + lane_off;
          mbar_wait(&s_full[buf], (Cfg::kSBufs == 2 ? tile_par : static_cast<uint32_t>(g / Cfg::kSBufs)) & 1);
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
          if (tail_tile(j)) {                                    // warp-uniform, last key tile of a ragged pass only
#pragma unroll
            for (int c = 0; c < kBlockN; ++c)
              if (c >= prm.k_tail) s[c] = 0xff800000u;           // -inf
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
            if (j > 0) {
              if (Cfg::kSBufs > 2) {     // the scores ran ahead of O_t += P_t(j-1) V: wait for it before touching O_t
                mbar_wait(&pv_done[t], tile_par ^ 1);
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
              const float2 p0 = ((Cfg::kPolyMask >> (i / 2)) & 1) ? ex2_poly2<kPolyDegree>(x0) : make_float2(ex2(x0.x), ex2(x0.y));
              const float2 p1 = ((Cfg::kPolyMask >> (i / 2 + 1)) & 1) ? ex2_poly2<kPolyDegree>(x1) : make_float2(ex2(x1.x), ex2(x1.y));
              la = fadd2(la, p0);
              lb = fadd2(lb, p1);
              pk[i / 2] = pack_bf16x2(p0.x, p0.y);
              pk[i / 2 + 1] = pack_bf16x2(p1.x, p1.y);
            }
            tmem_st_x16(tS + c * 16, pk);
            if (c & 1) {                       // 64 keys of P are in TMEM: let the tensor core start on them
              tmem_wait_st();
              tc_fence_before();
              if (Cfg::kSBufs > 2 && c == 1 && j > 0) mbar_wait(&pv_done[t], tile_par ^ 1);   // (see the split loop)
              mbar_arrive(&p_full[2 * t + (c >> 1)]);
            }
          }
          l += (la.x + la.y) + (lb.x + lb.y);
          g += 2;
          buf3 += 2;
          if (buf3 >= Cfg::kSBufs) buf3 -= Cfg::kSBufs;
          tile_par ^= 1;
        }
        mbar_wait(&o_full[t], li & 1);
      }
      // ---- chunk epilogue: loc_out = O / l, loc_lse = m*scale + ln l  (natural log of the scaled scores)
      // (O_t may be read here without further ado: the next item's first PV on this tile waits for P from these threads)
      tc_fence_after();
      float lse_row = (m_sc + lg2(l)) * 0.6931471805599453f;
      float cb = 1.0f / l, ca = 0.f;            // out = ca * o_acc + cb * O  (O = unnormalised accumulator in TMEM)
      if (kFold) {                              // Eq. 5, two operands: (o_acc, lse_acc) and (loc_out, loc_lse)
        // (in place, lse_out == lse_acc: both halves of a row read lse_acc at the item's start, half 0 overwrites it
        // below -- after the pair barrier of the row-sum exchange, which orders the partner's read before this write)
        const float m = fmaxf(lse_prev, lse_row);
        const float wa = ex2((lse_prev - m) * 1.4426950408889634f), wb = ex2((lse_row - m) * 1.4426950408889634f);
        const float den = wa + wb, r = 1.0f / den;
        ca = wa * r;
        cb *= wb * r;
        lse_row = m + lg2(den) * 0.6931471805599453f;
      }
      if (kOaccSmem) mbar_wait(oacc_full, li & 1);
#pragma unroll
      for (int c = 0; c < kD / 32; ++c) {
        if (Cfg::kColSplit && c / (kD / 64) != hh) continue;     // column split: each half stores its half of the row
        uint32_t o[32];
        tmem_ld_x32(tO + c * 32, o);
        float4 acc[8];
        if (kOaccSmem) {                          // panel (t, c): my row's 128 bytes, 16-byte chunks XOR-swizzled by row
          const uint8_t* prow = sOacc + (t * 2 + c) * Cfg::kPanelBytes + row_t * 128;
#pragma unroll
          for (int i = 0; i < 8; ++i) acc[i] = ld_shared_v4(prow + ((i ^ (row_t & 7)) << 4));
        } else if (kFold) {
          const float4* src = reinterpret_cast<const float4*>(prm.o_acc + acc_row * kD + c * 32);
#pragma unroll
          for (int i = 0; i < 8; ++i) acc[i] = row_valid() ? __ldcs(src + i) : make_float4(0.f, 0.f, 0.f, 0.f);
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
        if (!row_valid()) continue;
        if (kOutBf16) {
          uint4* dst = reinterpret_cast<uint4*>(static_cast<__nv_bfloat16*>(prm.o_out) + row * kD + c * 32);
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
          float4* dst = reinterpret_cast<float4*>(static_cast<float*>(prm.o_out) + row * kD + c * 32);
#pragma unroll
          for (int i = 0; i < 8; ++i) dst[i] = make_float4(r[i * 4], r[i * 4 + 1], r[i * 4 + 2], r[i * 4 + 3]);
        }
      }
      if (kOaccSmem) mbar_arrive(oacc_empty);        // my part of the o_acc tile is in registers / consumed
      if (hh == 0 && row_valid()) prm.lse_out[row] = lse_row;
      tc_fence_before();                             // my reads of O_t are ordered before the P I will signal next
      cur = next_item(li);
    }
  } else {
    setmaxnreg_dec<Cfg::kAuxRegs>();   // the idle warp of the last warpgroup: release its registers
  }

  tc_fence_before();
  __syncthreads();
  if (warp == Cfg::kProducerWarp) tmem_dealloc<512>(tmem);
}

template <int kD, int kEpi, bool kTail>
cudaError_t launch_tt(const CUtensorMap& mq, const CUtensorMap& mk, const CUtensorMap& mv, const CUtensorMap& moacc,
                      const FwdParams& prm, dim3 grid, cudaStream_t stream) {
  using Cfg = FwdCfg<kD>;
  auto kern = attn_chunk_fwd_kernel<kD, kEpi, kTail>;
  static unsigned char configured[kMaxDevices];
  if (cudaError_t e = set_max_dyn_smem_once(kern, Cfg::kSmemBytes, configured); e != cudaSuccess) return e;
  kern<<<grid, Cfg::kThreads, Cfg::kSmemBytes, stream>>>(mq, mk, mv, moacc, prm);
  count_launch();
  return cudaGetLastError();
}

template <int kD, int kEpi>
cudaError_t launch_t(const CUtensorMap& mq, const CUtensorMap& mk, const CUtensorMap& mv, const CUtensorMap& moacc,
                     const FwdParams& prm, dim3 grid, cudaStream_t stream) {
  if (prm.k_tail) return launch_tt<kD, kEpi, true>(mq, mk, mv, moacc, prm, grid, stream);
  return launch_tt<kD, kEpi, false>(mq, mk, mv, moacc, prm, grid, stream);
}

template <int kD>
cudaError_t launch_d(int epi, const CUtensorMap& mq, const CUtensorMap& mk, const CUtensorMap& mv, const CUtensorMap& moacc,
                     const FwdParams& prm, dim3 grid, cudaStream_t stream) {
  switch (epi) {
    case kEpiPartial:
      return launch_t<kD, kEpiPartial>(mq, mk, mv, moacc, prm, grid, stream);
    case kEpiFinal:
      return launch_t<kD, kEpiFinal>(mq, mk, mv, moacc, prm, grid, stream);
    case kEpiFold:
      return launch_t<kD, kEpiFold>(mq, mk, mv, moacc, prm, grid, stream);
    default:
      return launch_t<kD, kEpiFoldFinal>(mq, mk, mv, moacc, prm, grid, stream);
  }
}

}  // namespace

cudaError_t launch_attn_chunk_fwd_sm100(const void* q, const void* k, const void* v, void* o_out, float* lse_out,
                                        const float* o_acc, const float* lse_acc, int BH, int Nq, int nk_stride,
                                        int k_off, int nk, int d, float scale, int epilogue, int splits,
                                        cudaStream_t stream) {
  const int n_tiles = (nk + kBlockN - 1) / kBlockN;      // the last one may be ragged (then k_off + nk == nk_stride)
  if (splits < 1 || (splits > 1 && (epilogue != kFwdEpiPartial || nk % kBlockN)) || n_tiles % splits) return cudaErrorInvalidValue;
  if (nk % kBlockN && k_off + nk != nk_stride) return cudaErrorInvalidValue;
  CUtensorMap mq, mk, mv, moacc;
  const CUtensorMapDataType dt = CU_TENSOR_MAP_DATA_TYPE_BFLOAT16;
  // [BH][rows][d] views: a tile that runs past the end of a head reads zeros there, not the next head's rows
  if (!make_tmap_3d(&mq, q, dt, 2, BH, Nq, d, 128, 64, kSwizzle128B) ||
      !make_tmap_3d(&mk, k, dt, 2, BH, nk_stride, d, 128, 64, kSwizzle128B) ||
      !make_tmap_3d(&mv, v, dt, 2, BH, nk_stride, d, 128, 64, kSwizzle128B))
    return cudaErrorInvalidValue;
  const bool fold = epilogue == kFwdEpiFold || epilogue == kFwdEpiFoldFinal;
  moacc = mq;                                  // (unused unless d = 64 and the epilogue folds)
  if (fold && d == 64 &&
      !make_tmap_3d(&moacc, o_acc, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, BH, Nq, d, 128, 32, kSwizzle128B))
    return cudaErrorInvalidValue;
  FwdParams prm;
  prm.o_out = o_out;
  prm.lse_out = lse_out;
  prm.o_acc = o_acc;
  prm.lse_acc = lse_acc;
  prm.Nq = Nq;
  prm.nk_stride = nk_stride;
  prm.k_off = k_off;
  prm.n_kv = n_tiles / splits;
  prm.k_tail = nk % kBlockN;
  prm.scale_log2 = scale * 1.4426950408889634f;
  const dim3 grid((Nq + 2 * kBlockM - 1) / (2 * kBlockM), BH, splits);      // one CTA per item; most are cancelled and taken over (see the top)
  if (d == 64) return launch_d<64>(epilogue, mq, mk, mv, moacc, prm, grid, stream);
  return launch_d<128>(epilogue, mq, mk, mv, moacc, prm, grid, stream);
}

}  // namespace ringx
