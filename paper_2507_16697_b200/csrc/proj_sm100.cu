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
  int M, N, K;      // GEMM extents: M = B*S, N = 3h (QKV) or h (OUT), K = h
  int S, H, d, h;   // head-split geometry
  int m_tiles, n_tiles;
};

template <int kMode>   // 0 = QKV, 1 = OUT
__global__ void __launch_bounds__(kProjThreads, 1)
proj_gemm_kernel(const __grid_constant__ CUtensorMap map_a, const __grid_constant__ CUtensorMap map_b,
                 const __grid_constant__ CUtensorMap map_c0, const __grid_constant__ CUtensorMap map_c1,
                 const __grid_constant__ CUtensorMap map_c2, const ProjParams p) {
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
  const int n_tiles_total = p.m_tiles * p.n_tiles;
  const int k_blocks = p.K / kBK;

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
      prefetch_tmap(&map_a);
      prefetch_tmap(&map_b);
      prefetch_tmap(&map_c0);
      if (kMode == 0) {
        prefetch_tmap(&map_c1);
        prefetch_tmap(&map_c2);
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
    const uint64_t pol_a = policy_evict_first(), pol_b = policy_evict_last();   // W is re-read by every CTA
    int st = 0, ph = 0;
    for (int t = blockIdx.x; t < n_tiles_total; t += gridDim.x) {
      const int m0 = (t / p.n_tiles) * kBM, n0 = (t % p.n_tiles) * kBN;
      for (int kb = 0; kb < k_blocks; ++kb) {
        mbar_wait_relaxed(&empty[st], ph ^ 1);
        if (leader) {
          uint8_t* dst = sStage + st * kStageBytes;
          mbar_arrive_expect_tx(&full[st], kStageBytes);
          int a_col = kb * kBK, a_row = m0;
          if (kMode == 1) {   // A = o in [B,H,S,d]: this K block is 64 features of head (kb*64)/d
            const int head = a_col / p.d, b = m0 / p.S, s0 = m0 - b * p.S;
            a_row = (b * p.H + head) * p.S + s0;
            a_col -= head * p.d;
          }
          tma_load_2d(dst, &map_a, &full[st], a_col, a_row, pol_a);
          tma_load_2d(dst + kABytes, &map_b, &full[st], kb * kBK, n0, pol_b);
        }
        __syncwarp();
        if (++st == kStages) { st = 0; ph ^= 1; }
      }
    }
  } else if (warp == 1) {
    // ---------------------------------------------------------------- MMA issuer
    const bool leader = elect_one();
    constexpr uint32_t idesc = make_idesc_bf16(kBM, kBN, 0, 0);
    const uint32_t stage_base = smem_u32(sStage);
    int st = 0, ph = 0, it = 0;
    for (int t = blockIdx.x; t < n_tiles_total; t += gridDim.x, ++it) {
      const int ab = it & 1;
      mbar_wait(&acc_empty[ab], ((it >> 1) & 1) ^ 1);          // the epilogue has drained this accumulator
      tc_fence_after();
      const uint32_t acc = tmem + ab * kBN;
      for (int kb = 0; kb < k_blocks; ++kb) {
        mbar_wait(&full[st], ph);
        tc_fence_after();
        if (leader) {
          const uint32_t a_addr = stage_base + st * kStageBytes, b_addr = a_addr + kABytes;
#pragma unroll
          for (int k = 0; k < kBK / 16; ++k)
            mma_ss(acc, make_smem_desc_sw128(a_addr + k * 32, 16, 1024), make_smem_desc_sw128(b_addr + k * 32, 16, 1024),
                   idesc, kb > 0 || k > 0);
          mma_commit(&empty[st]);
          if (kb == k_blocks - 1) mma_commit(&acc_full[ab]);
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
    int it = 0, buf = 0;
    for (int t = blockIdx.x; t < n_tiles_total; t += gridDim.x, ++it) {
      const int ab = it & 1;
      const int m0 = (t / p.n_tiles) * kBM, n0 = (t % p.n_tiles) * kBN;
      mbar_wait(&acc_full[ab], (it >> 1) & 1);
      tc_fence_after();
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
          if (kMode == 0) {   // column n of [q|k|v]: tensor n / h, head (n % h) / d, feature n % d
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

int sm_count() {
  static int n = 0;
  if (!n) {
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev);
  }
  return n;
}

template <int kMode>
cudaError_t launch_mode(const CUtensorMap& ma, const CUtensorMap& mb, const CUtensorMap& c0, const CUtensorMap& c1,
                        const CUtensorMap& c2, const ProjParams& p, cudaStream_t stream) {
  auto kern = proj_gemm_kernel<kMode>;
  static bool configured = false;
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kProjSmem);
    if (e != cudaSuccess) return e;
    configured = true;
  }
  const int tiles = p.m_tiles * p.n_tiles;
  const int grid = tiles < sm_count() ? tiles : sm_count();
  kern<<<grid, kProjThreads, kProjSmem, stream>>>(ma, mb, c0, c1, c2, p);
  count_launch();
  return cudaGetLastError();
}

}  // namespace

// x [B,S,h], w_qkv [3h,h] -> q,k,v [B,H,S,d] (all bf16)
cudaError_t launch_qkv_proj(const void* x, const void* w_qkv, void* q, void* k, void* v, int B, int S, int H, int d,
                            cudaStream_t stream) {
  const int h = H * d;
  const CUtensorMapDataType dt = CU_TENSOR_MAP_DATA_TYPE_BFLOAT16;
  CUtensorMap ma, mb, c0, c1, c2;
  const uint64_t M = (uint64_t)B * S;
  if (!make_tmap_2d(&ma, x, dt, 2, M, h, kBM, kBK, kSwizzle128B) ||
      !make_tmap_2d(&mb, w_qkv, dt, 2, 3ull * h, h, kBN, kBK, kSwizzle128B) ||
      !make_tmap_2d(&c0, q, dt, 2, M * H, d, 128, 64, kSwizzle128B) ||
      !make_tmap_2d(&c1, k, dt, 2, M * H, d, 128, 64, kSwizzle128B) ||
      !make_tmap_2d(&c2, v, dt, 2, M * H, d, 128, 64, kSwizzle128B))
    return cudaErrorInvalidValue;
  ProjParams p{(int)M, 3 * h, h, S, H, d, h, (int)(M / kBM), (3 * h + kBN - 1) / kBN};
  return launch_mode<0>(ma, mb, c0, c1, c2, p, stream);
}

// o [B,H,S,d], w_o [h,h] -> y [B,S,h] (all bf16)
cudaError_t launch_out_proj(const void* o, const void* w_o, void* y, int B, int S, int H, int d, cudaStream_t stream) {
  const int h = H * d;
  const CUtensorMapDataType dt = CU_TENSOR_MAP_DATA_TYPE_BFLOAT16;
  CUtensorMap ma, mb, c0;
  const uint64_t M = (uint64_t)B * S;
  if (!make_tmap_2d(&ma, o, dt, 2, M * H, d, kBM, kBK, kSwizzle128B) ||
      !make_tmap_2d(&mb, w_o, dt, 2, h, h, kBN, kBK, kSwizzle128B) ||
      !make_tmap_2d(&c0, y, dt, 2, M, h, 128, 64, kSwizzle128B))
    return cudaErrorInvalidValue;
  ProjParams p{(int)M, h, h, S, H, d, h, (int)(M / kBM), (h + kBN - 1) / kBN};
  return launch_mode<1>(ma, mb, c0, c0, c0, p, stream);
}

}  // namespace ringx
