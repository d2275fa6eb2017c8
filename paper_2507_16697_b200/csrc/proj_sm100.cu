// proj_sm100.cu -- the projection GEMMs either side of the attention kernel (Table II), on tcgen05:
//   mode QKV : [q|k|v] = x W_qkv^T, written straight into the head-split layout (b*a, S, h/a) the attention kernels read
//   mode OUT : y = merge_heads(o) W_o^T, reading o in the head-split layout
// C[M, N] = A[M, K] B[N, K]^T, bf16 operands (both K-major), fp32 accumulation in TMEM, bf16 output.  The head split /
// merge costs nothing: a 64-column block of C (or a 64-element K block of A) lies inside one head, so it is just a
// different TMA coordinate -- no transpose kernel, no extra pass over HBM.
//
// Persistent CTAs (one per SM), tile 128 x 256, K blocks of 64 (one 128-byte-swizzled panel):
//   warp 0      TMA producer: A [128 x 64] + B [256 x 64] per stage, 4-stage ring
//   warp 1      MMA issuer: 4 x tcgen05.mma M128 N256 K16 per stage into one of two TMEM accumulators (2 x 256 columns)
//   warps 2-5   epilogue: TMEM -> registers -> bf16 -> 128B-swizzled staging panel [128 x 64] -> TMA store; runs under
//               the next tile's main loop (double-buffered accumulator)
// Ragged N (N % 256 != 0, N % 64 == 0): TMA zero-fills the out-of-range B rows; the epilogue skips their columns.
#include "kernels.cuh"

namespace ringx {
namespace {

using namespace ptx;

constexpr int kBM = 128, kBN = 256, kBK = 64;
constexpr int kStages = 4;
constexpr int kABytes = kBM * kBK * 2, kBBytes = kBN * kBK * 2, kStageBytes = kABytes + kBBytes;
constexpr int kPanelBytes = 128 * 128;                       // one [128 x 64] bf16 staging panel
constexpr int kProjSmem = 1024 + kStages * kStageBytes + 2 * kPanelBytes + 256;
constexpr int kProjThreads = 192;

struct ProjParams {
  int M, N, K;      // GEMM extents (rows of C, columns of C, reduction length)
  int S, H, d, h;   // head-split geometry
  int m_tiles, n_tiles;
  int splits;       // split-K factor (weight-gradient modes; 1 otherwise)
  int kb_per;       // K blocks per split
};

// Modes.  "head-split" operands live in [B,H,S,d] tensors viewed as [B*H*S, d]; a 64-wide block of merged features
// lies inside one head, so merging / splitting heads is a TMA coordinate, never a transpose pass.
//   0 QKV forward        [q|k|v] = x W_qkv^T          A x K-major          B W_qkv K-major      C bf16 head-split (3 tensors)
//   1 OUT forward        y = merge(o) W_o^T           A o head-merged      B W_o K-major        C bf16 plain
//   2 OUT data grad      dO = split(dY W_o)           A dY K-major         B W_o MN-major       C bf16 head-split (1 tensor)
//   3 QKV data grad      dX = merge[dq|dk|dv] W_qkv   A dq,dk,dv merged    B W_qkv MN-major     C bf16 plain
//   4 OUT weight grad    dW_o = dY^T merge(o)         A dY MN-major        B o merged MN-major  C fp32 reduce-add, split-K
//   5 QKV weight grad    dW_qkv = merge[..]^T x       A dq,dk,dv MN-major  B x MN-major         C fp32 reduce-add, split-K
template <int kMode>
struct ProjMode {
  static constexpr bool kAMn = kMode >= 4, kBMn = kMode >= 2;
  static constexpr bool kOutF32 = kMode >= 4;
  static constexpr bool kOutHeadSplit = kMode == 0 || kMode == 2;
};
constexpr int kMnPanelBytes = 64 * 128;    // MN-major operand panel: 64 K-rows x 64 MN-elements (128 B)

template <int kMode>
__global__ void __launch_bounds__(kProjThreads, 1)
proj_gemm_kernel(const __grid_constant__ CUtensorMap map_a0, const __grid_constant__ CUtensorMap map_a1,
                 const __grid_constant__ CUtensorMap map_a2, const __grid_constant__ CUtensorMap map_b,
                 const __grid_constant__ CUtensorMap map_c0, const __grid_constant__ CUtensorMap map_c1,
                 const __grid_constant__ CUtensorMap map_c2, const ProjParams p) {
  using Md = ProjMode<kMode>;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t* sStage = smem;
  uint8_t* sOut = smem + kStages * kStageBytes;
  uint64_t* bars = reinterpret_cast<uint64_t*>(sOut + 2 * kPanelBytes);
  uint64_t* full = bars;                  // [kStages] TMA -> MMA
  uint64_t* empty = bars + kStages;       // [kStages] MMA -> TMA
  uint64_t* acc_full = bars + 2 * kStages;     // [2] MMA -> epilogue
  uint64_t* acc_empty = acc_full + 2;          // [2] epilogue -> MMA   (128 arrivals)
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(acc_empty + 2);

  const int warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0);
  const int lane = threadIdx.x & 31;
  const int n_items = p.m_tiles * p.n_tiles * p.splits;
  const int k_blocks = p.K / kBK;
  // item -> (tile, split); the split index is fastest so that the CTAs working on one tile run concurrently
  auto item_tile = [&](int it, int& m0, int& n0, int& kb0, int& kb1) {
    const int split = it % p.splits, tile = it / p.splits;
    m0 = (tile / p.n_tiles) * kBM;
    n0 = (tile % p.n_tiles) * kBN;
    kb0 = split * p.kb_per;
    kb1 = kb0 + p.kb_per < k_blocks ? kb0 + p.kb_per : k_blocks;
  };

  if (threadIdx.x == 0) {
    for (int i = 0; i < kStages; ++i) {
      mbar_init(&full[i], 1);
      mbar_init(&empty[i], 1);
    }
    for (int i = 0; i < 2; ++i) {
      mbar_init(&acc_full[i], 1);
      mbar_init(&acc_empty[i], 128);
    }
    fence_mbar_init();
  }
  if (warp == 0) {
    if (lane == 0) {
      prefetch_tmap(&map_a0);
      prefetch_tmap(&map_b);
      prefetch_tmap(&map_c0);
      if (kMode == 0) {
        prefetch_tmap(&map_c1);
        prefetch_tmap(&map_c2);
      }
      if (kMode == 3 || kMode == 5) {
        prefetch_tmap(&map_a1);
        prefetch_tmap(&map_a2);
      }
    }
    tmem_alloc<512>(tmem_slot);
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_slot;

  if (warp == 0) {
    // ---------------------------------------------------------------- TMA producer
    const bool leader = elect_one();
    const uint64_t pol_stream = policy_evict_first(), pol_keep = policy_evict_last();
    // the operand every CTA re-reads (the weights in modes 0-3) stays in L2; activations stream
    const uint64_t pol_a = pol_stream, pol_b = kMode <= 3 ? pol_keep : pol_stream;
    // row of token (b, s0) of head `head` in a [B*H*S, d] view, for the merged feature column f (head = f / d)
    auto head_row = [&](int token, int head) {
      const int b = token / p.S;
      return (b * p.H + head) * p.S + (token - b * p.S);
    };
    int st = 0, ph = 0;
    for (int it = blockIdx.x; it < n_items; it += gridDim.x) {
      int m0, n0, kb0, kb1;
      item_tile(it, m0, n0, kb0, kb1);
      for (int kb = kb0; kb < kb1; ++kb) {
        mbar_wait_relaxed(&empty[st], ph ^ 1);
        if (leader) {
          uint8_t* dst = sStage + st * kStageBytes;
          const int k0 = kb * kBK;
          mbar_arrive_expect_tx(&full[st], kStageBytes);
          // ---- A
          if (kMode == 0 || kMode == 2) {
            tma_load_2d(dst, &map_a0, &full[st], k0, m0, pol_a);
          } else if (kMode == 1 || kMode == 3) {          // K block = 64 merged features of one head (of one of q,k,v)
            const int which = k0 / p.h, f = k0 - which * p.h, head = f / p.d;
            const CUtensorMap* ma = which == 0 ? &map_a0 : which == 1 ? &map_a1 : &map_a2;
            tma_load_2d(dst, ma, &full[st], f - head * p.d, head_row(m0, head), pol_a);
          } else {                                        // MN-major: two panels of 64 C-rows x 64 tokens
#pragma unroll
            for (int pn = 0; pn < kBM / 64; ++pn) {
              const int col = m0 + pn * 64;
              if (kMode == 4) {
                tma_load_2d(dst + pn * kMnPanelBytes, &map_a0, &full[st], col, k0, pol_a);
              } else {
                const int which = col / p.h, f = col - which * p.h, head = f / p.d;
                const CUtensorMap* ma = which == 0 ? &map_a0 : which == 1 ? &map_a1 : &map_a2;
                tma_load_2d(dst + pn * kMnPanelBytes, ma, &full[st], f - head * p.d, head_row(k0, head), pol_a);
              }
            }
          }
          // ---- B
          if (!Md::kBMn) {
            tma_load_2d(dst + kABytes, &map_b, &full[st], k0, n0, pol_b);
          } else {
#pragma unroll
            for (int pn = 0; pn < kBN / 64; ++pn) {
              const int col = n0 + pn * 64;
              if (kMode == 4) {                           // o, head-merged
                const int head = col / p.d;
                tma_load_2d(dst + kABytes + pn * kMnPanelBytes, &map_b, &full[st], col - head * p.d, head_row(k0, head), pol_b);
              } else {
                tma_load_2d(dst + kABytes + pn * kMnPanelBytes, &map_b, &full[st], col, k0, pol_b);
              }
            }
          }
        }
        __syncwarp();
        if (++st == kStages) { st = 0; ph ^= 1; }
      }
    }
  } else if (warp == 1) {
    // ---------------------------------------------------------------- MMA issuer
    const bool leader = elect_one();
    constexpr uint32_t idesc = make_idesc_bf16(kBM, kBN, Md::kAMn ? 1 : 0, Md::kBMn ? 1 : 0);
    const uint32_t stage_base = smem_u32(sStage);
    int st = 0, ph = 0, n = 0;
    for (int it = blockIdx.x; it < n_items; it += gridDim.x, ++n) {
      int m0, n0, kb0, kb1;
      item_tile(it, m0, n0, kb0, kb1);
      const int ab = n & 1;
      mbar_wait(&acc_empty[ab], ((n >> 1) & 1) ^ 1);          // the epilogue has drained this accumulator
      tc_fence_after();
      const uint32_t acc = tmem + ab * kBN;
      for (int kb = kb0; kb < kb1; ++kb) {
        mbar_wait(&full[st], ph);
        tc_fence_after();
        if (leader) {
          const uint32_t a_addr = stage_base + st * kStageBytes, b_addr = a_addr + kABytes;
#pragma unroll
          for (int k = 0; k < kBK / 16; ++k) {
            const uint64_t da = Md::kAMn ? make_smem_desc_sw128(a_addr + k * 2048, kMnPanelBytes, 1024)
                                         : make_smem_desc_sw128(a_addr + k * 32, 16, 1024);
            const uint64_t db = Md::kBMn ? make_smem_desc_sw128(b_addr + k * 2048, kMnPanelBytes, 1024)
                                         : make_smem_desc_sw128(b_addr + k * 32, 16, 1024);
            mma_ss(acc, da, db, idesc, kb > kb0 || k > 0);
          }
          mma_commit(&empty[st]);
          if (kb == kb1 - 1) mma_commit(&acc_full[ab]);
        }
        __syncwarp();
        if (++st == kStages) { st = 0; ph ^= 1; }
      }
    }
  } else {
    // ---------------------------------------------------------------- epilogue warps (2-5): thread = output row
    const int lane_grp = warp & 3;                               // tcgen05.ld: warp w may touch lanes 32*(w%4)..+31
    const int row = lane_grp * 32 + lane;
    const uint32_t lane_off = static_cast<uint32_t>(lane_grp * 32) << 16;
    const bool leader = warp == 2 && elect_one();
    int n_it = 0, buf = 0;
    for (int it = blockIdx.x; it < n_items; it += gridDim.x, ++n_it) {
      int m0, n0, kb0, kb1;
      item_tile(it, m0, n0, kb0, kb1);
      const int ab = n_it & 1;
      mbar_wait(&acc_full[ab], (n_it >> 1) & 1);
      tc_fence_after();
      if (Md::kOutF32) {
        // fp32 partial sums of this K split, reduce-added into C by TMA (32 columns = one 128-byte swizzled panel)
#pragma unroll 1
        for (int c = 0; c < kBN / 32; ++c) {
          uint32_t r0[32];
          tmem_ld_x32(tmem + ab * kBN + lane_off + c * 32, r0);
          tmem_wait_ld_x32(r0);
          if (leader) tma_wait_group_read<1>();
          named_bar_sync(1, 128);
          uint8_t* prow = sOut + buf * kPanelBytes + row * 128;
#pragma unroll
          for (int g = 0; g < 8; ++g)
            st_shared_v4(prow + ((g ^ (row & 7)) << 4), r0[g * 4], r0[g * 4 + 1], r0[g * 4 + 2], r0[g * 4 + 3]);
          fence_proxy_async_smem();
          named_bar_sync(2, 128);
          if (leader) {
            tma_reduce_add_2d(&map_c0, sOut + buf * kPanelBytes, n0 + c * 32, m0);
            tma_commit_group();
          }
          buf ^= 1;
        }
      } else {
#pragma unroll 1
        for (int c = 0; c < kBN / 64; ++c) {
          const int n = n0 + c * 64;
          if (n >= p.N) break;                                     // ragged last N tile
          uint32_t r0[32], r1[32];
          tmem_ld_x32(tmem + ab * kBN + lane_off + c * 64, r0);
          tmem_ld_x32(tmem + ab * kBN + lane_off + c * 64 + 32, r1);
          tmem_wait_ld_x32(r0);
          tmem_wait_ld_x32(r1);
          if (leader) tma_wait_group_read<1>();                    // the store that last read this panel is done with it
          named_bar_sync(1, 128);
          uint8_t* prow = sOut + buf * kPanelBytes + row * 128;
#pragma unroll
          for (int g = 0; g < 4; ++g)
            st_shared_v4(prow + ((g ^ (row & 7)) << 4),
                         pack_bf16x2(__uint_as_float(r0[g * 8 + 0]), __uint_as_float(r0[g * 8 + 1])),
                         pack_bf16x2(__uint_as_float(r0[g * 8 + 2]), __uint_as_float(r0[g * 8 + 3])),
                         pack_bf16x2(__uint_as_float(r0[g * 8 + 4]), __uint_as_float(r0[g * 8 + 5])),
                         pack_bf16x2(__uint_as_float(r0[g * 8 + 6]), __uint_as_float(r0[g * 8 + 7])));
#pragma unroll
          for (int g = 0; g < 4; ++g)
            st_shared_v4(prow + (((g + 4) ^ (row & 7)) << 4),
                         pack_bf16x2(__uint_as_float(r1[g * 8 + 0]), __uint_as_float(r1[g * 8 + 1])),
                         pack_bf16x2(__uint_as_float(r1[g * 8 + 2]), __uint_as_float(r1[g * 8 + 3])),
                         pack_bf16x2(__uint_as_float(r1[g * 8 + 4]), __uint_as_float(r1[g * 8 + 5])),
                         pack_bf16x2(__uint_as_float(r1[g * 8 + 6]), __uint_as_float(r1[g * 8 + 7])));
          fence_proxy_async_smem();
          named_bar_sync(2, 128);
          if (leader) {
            if (Md::kOutHeadSplit) {   // column n of [q|k|v] (or of dO): tensor n / h, head (n % h) / d, feature n % d
              const int which = n / p.h, f = n - which * p.h, head = f / p.d;
              const int b = m0 / p.S, s0 = m0 - b * p.S;
              const CUtensorMap* mc = which == 0 ? &map_c0 : which == 1 ? &map_c1 : &map_c2;
              tma_store_2d(mc, sOut + buf * kPanelBytes, f - head * p.d, (b * p.H + head) * p.S + s0);
            } else {
              tma_store_2d(&map_c0, sOut + buf * kPanelBytes, n, m0);
            }
            tma_commit_group();
          }
          buf ^= 1;
        }
      }
      tc_fence_before();
      mbar_arrive(&acc_empty[ab]);                               // all my TMEM reads of this accumulator are done
    }
    if (leader) tma_wait_group<0>();
    __syncwarp();
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc<512>(tmem);
}

template <int kMode>
cudaError_t launch_mode(const CUtensorMap& a0, const CUtensorMap& a1, const CUtensorMap& a2, const CUtensorMap& mb,
                        const CUtensorMap& c0, const CUtensorMap& c1, const CUtensorMap& c2, const ProjParams& p,
                        cudaStream_t stream) {
  auto kern = proj_gemm_kernel<kMode>;
  static unsigned char configured[kMaxDevices];
  if (cudaError_t e = set_max_dyn_smem_once(kern, kProjSmem, configured); e != cudaSuccess) return e;
  const int items = p.m_tiles * p.n_tiles * p.splits;
  const int grid = items < sm_count() ? items : sm_count();
  kern<<<grid, kProjThreads, kProjSmem, stream>>>(a0, a1, a2, mb, c0, c1, c2, p);
  count_launch();
  return cudaGetLastError();
}

constexpr CUtensorMapDataType kBf16 = CU_TENSOR_MAP_DATA_TYPE_BFLOAT16;

// K-major operand tile: box = 64 reduction elements x `rows` rows; MN-major operand panel: 64 x 64
bool tmap_kmajor(CUtensorMap* m, const void* base, uint64_t rows, uint64_t cols, uint32_t box_rows) {
  return make_tmap_2d(m, base, kBf16, 2, rows, cols, box_rows, kBK, kSwizzle128B);
}
bool tmap_mnmajor(CUtensorMap* m, const void* base, uint64_t rows, uint64_t cols) {
  return make_tmap_2d(m, base, kBf16, 2, rows, cols, 64, 64, kSwizzle128B);
}
bool tmap_out_bf16(CUtensorMap* m, void* base, uint64_t rows, uint64_t cols) {
  return make_tmap_2d(m, base, kBf16, 2, rows, cols, 128, 64, kSwizzle128B);
}
bool tmap_out_f32(CUtensorMap* m, void* base, uint64_t rows, uint64_t cols) {
  return make_tmap_2d(m, base, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, rows, cols, 128, 32, kSwizzle128B);
}

ProjParams make_params(long long M, int N, long long K, int S, int H, int d, bool split_k) {
  ProjParams p{};
  p.M = (int)M; p.N = N; p.K = (int)K;
  p.S = S; p.H = H; p.d = d; p.h = H * d;
  p.m_tiles = (int)((M + kBM - 1) / kBM);
  p.n_tiles = (N + kBN - 1) / kBN;
  const int k_blocks = (int)(K / kBK);
  p.splits = 1;
  p.kb_per = k_blocks;
  if (split_k) {      // few output tiles, a long reduction: split it so that ~2 waves of CTAs have work
    int want = (2 * sm_count()) / (p.m_tiles * p.n_tiles);
    if (want < 1) want = 1;
    if (want > k_blocks) want = k_blocks;
    p.kb_per = (k_blocks + want - 1) / want;
    p.splits = (k_blocks + p.kb_per - 1) / p.kb_per;      // no empty split
  }
  return p;
}

}  // namespace

// x [B,S,h], w_qkv [3h,h] -> q,k,v [B,H,S,d] (all bf16)
cudaError_t launch_qkv_proj(const void* x, const void* w_qkv, void* q, void* k, void* v, int B, int S, int H, int d,
                            cudaStream_t stream) {
  const int h = H * d;
  CUtensorMap ma, mb, c0, c1, c2;
  const uint64_t M = (uint64_t)B * S;
  if (!tmap_kmajor(&ma, x, M, h, kBM) || !tmap_kmajor(&mb, w_qkv, 3ull * h, h, kBN) || !tmap_out_bf16(&c0, q, M * H, d) ||
      !tmap_out_bf16(&c1, k, M * H, d) || !tmap_out_bf16(&c2, v, M * H, d))
    return cudaErrorInvalidValue;
  return launch_mode<0>(ma, ma, ma, mb, c0, c1, c2, make_params(M, 3 * h, h, S, H, d, false), stream);
}

// o [B,H,S,d], w_o [h,h] -> y [B,S,h] (all bf16)
cudaError_t launch_out_proj(const void* o, const void* w_o, void* y, int B, int S, int H, int d, cudaStream_t stream) {
  const int h = H * d;
  CUtensorMap ma, mb, c0;
  const uint64_t M = (uint64_t)B * S;
  if (!tmap_kmajor(&ma, o, M * H, d, kBM) || !tmap_kmajor(&mb, w_o, h, h, kBN) || !tmap_out_bf16(&c0, y, M, h))
    return cudaErrorInvalidValue;
  return launch_mode<1>(ma, ma, ma, mb, c0, c0, c0, make_params(M, h, h, S, H, d, false), stream);
}

// dy [B,S,h], o [B,H,S,d], w_o [h,h] -> d_o [B,H,S,d] bf16, dw_o [h,h] fp32 (zeroed by the caller, reduce-added here)
cudaError_t launch_out_proj_bwd(const void* dy, const void* o, const void* w_o, void* d_o, float* dw_o, int B, int S,
                                int H, int d, cudaStream_t stream) {
  const int h = H * d;
  const uint64_t M = (uint64_t)B * S;
  CUtensorMap ma, mb, c0;
  // dO = split(dY W_o): A = dY K-major, B = W_o as [K = n rows][N = i contiguous] (MN-major)
  if (!tmap_kmajor(&ma, dy, M, h, kBM) || !tmap_mnmajor(&mb, w_o, h, h) || !tmap_out_bf16(&c0, d_o, M * H, d))
    return cudaErrorInvalidValue;
  cudaError_t e = launch_mode<2>(ma, ma, ma, mb, c0, c0, c0, make_params(M, h, h, S, H, d, false), stream);
  if (e != cudaSuccess) return e;
  // dW_o[n,i] = sum_m dY[m,n] o_merged[m,i]: both operands MN-major (the token index m is the reduction)
  if (!tmap_mnmajor(&ma, dy, M, h) || !tmap_mnmajor(&mb, o, M * H, d) || !tmap_out_f32(&c0, dw_o, h, h))
    return cudaErrorInvalidValue;
  return launch_mode<4>(ma, ma, ma, mb, c0, c0, c0, make_params(h, h, (long long)M, S, H, d, true), stream);
}

// dq,dk,dv [B,H,S,d], x [B,S,h], w_qkv [3h,h] -> dx [B,S,h] bf16, dw_qkv [3h,h] fp32 (zeroed by the caller)
cudaError_t launch_qkv_proj_bwd(const void* dq, const void* dk, const void* dv, const void* x, const void* w_qkv,
                                void* dx, float* dw_qkv, int B, int S, int H, int d, cudaStream_t stream) {
  const int h = H * d;
  const uint64_t M = (uint64_t)B * S;
  CUtensorMap a0, a1, a2, mb, c0;
  // dX = merge[dq|dk|dv] W_qkv: A = head-merged K-major (K = 3h), B = W_qkv as [K = n rows][N = i contiguous]
  if (!tmap_kmajor(&a0, dq, M * H, d, kBM) || !tmap_kmajor(&a1, dk, M * H, d, kBM) || !tmap_kmajor(&a2, dv, M * H, d, kBM) ||
      !tmap_mnmajor(&mb, w_qkv, 3ull * h, h) || !tmap_out_bf16(&c0, dx, M, h))
    return cudaErrorInvalidValue;
  cudaError_t e = launch_mode<3>(a0, a1, a2, mb, c0, c0, c0, make_params(M, h, 3LL * h, S, H, d, false), stream);
  if (e != cudaSuccess) return e;
  // dW_qkv[n,i] = sum_m merge[dq|dk|dv][m,n] x[m,i]
  if (!tmap_mnmajor(&a0, dq, M * H, d) || !tmap_mnmajor(&a1, dk, M * H, d) || !tmap_mnmajor(&a2, dv, M * H, d) ||
      !tmap_mnmajor(&mb, x, M, h) || !tmap_out_f32(&c0, dw_qkv, 3ull * h, h))
    return cudaErrorInvalidValue;
  return launch_mode<5>(a0, a1, a2, mb, c0, c0, c0, make_params(3LL * h, h, (long long)M, S, H, d, true), stream);
}

}  // namespace ringx
