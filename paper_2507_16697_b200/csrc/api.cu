// api.cu -- the C-ABI layer of libringx (include/ringx.h): argument validation, workspace carving,
// TMA tensor-map creation and the KV-chunk pass loop.  No arithmetic of the method lives here; every
// step of the path runs in the kernels this file launches.
#include <math.h>

#include <atomic>
#include <mutex>
#include <vector>

#include "kernels.cuh"

namespace ringx {

namespace {

thread_local int tl_launches = 0;
thread_local int tl_last_launches = 0;

constexpr size_t kAlign = 256;
inline size_t align_up(size_t x) { return (x + kAlign - 1) / kAlign * kAlign; }
inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

using EncodeFn = CUresult (*)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                              const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                              CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeFn encode_fn() {
  static EncodeFn fn = nullptr;
  static std::once_flag once;
  std::call_once(once, [] {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult qr;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qr) == cudaSuccess &&
        qr == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<EncodeFn>(p);
  });
  return fn;
}

// RINGX_OK when the current device is compute capability 10.x.
int check_arch() {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) {
    cudaGetLastError();
    return RINGX_ERR_CUDA;
  }
  static std::mutex mu;
  static int cached[kMaxDevices];   // 0 = unknown, 1 = ok, 2 = unsupported
  std::lock_guard<std::mutex> g(mu);
  if (dev >= 0 && dev < kMaxDevices && cached[dev]) return cached[dev] == 1 ? RINGX_OK : RINGX_ERR_UNSUPPORTED_ARCH;
  int major = 0;
  if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) {
    cudaGetLastError();
    return RINGX_ERR_CUDA;
  }
  if (dev >= 0 && dev < kMaxDevices) cached[dev] = (major == 10) ? 1 : 2;
  return major == 10 ? RINGX_OK : RINGX_ERR_UNSUPPORTED_ARCH;
}

// `ragged_ok`: the entry point takes any sequence length (bf16 ringx_attn_fwd / ringx_attn_bwd and their GQA forms): the
// kernels zero-fill and mask what lies past the end of a head, and the last KV chunk may be shorter than kv_chunk.
int check_shape(int B, int H, int N, int d, int kv_chunk, float scale, int dtype, bool backward, bool ragged_ok = false) {
  if (dtype != RINGX_F32 && dtype != RINGX_BF16) return RINGX_ERR_BAD_DTYPE;
  if (backward && dtype != RINGX_BF16) return RINGX_ERR_BAD_DTYPE;
  if (B <= 0 || H <= 0 || N <= 0 || kv_chunk <= 0) return RINGX_ERR_BAD_SHAPE;
  if (d != 64 && d != 128) return RINGX_ERR_BAD_SHAPE;
  if (kv_chunk % 128) return RINGX_ERR_BAD_SHAPE;
  if (ragged_ok && dtype == RINGX_BF16) {
    if (kv_chunk > (N + 127) / 128 * 128) return RINGX_ERR_BAD_SHAPE;
  } else {
    if (N % 128 || kv_chunk > N || N % kv_chunk) return RINGX_ERR_BAD_SHAPE;
    if (dtype == RINGX_BF16 && !backward && N % 256) return RINGX_ERR_BAD_SHAPE;
  }
  if ((long long)B * H > 65535) return RINGX_ERR_BAD_SHAPE;
  if ((long long)B * H * N > 0x7FFFFFFFLL) return RINGX_ERR_BAD_SHAPE;   // TMA row coordinate is int32
  if (!(scale > 0.f) || !(scale < 3.0e38f)) return RINGX_ERR_BAD_SHAPE;
  return RINGX_OK;
}

// ---- split-KV: when one chunk pass has too few query tiles to fill the GPU (the paper's own regime: 2K-64K query tokens per
// device against a long gathered key sequence), the keys of the pass are split over gridDim.z and the
// splits' partials are combined by Eq. 5 -- the same merge, inside one pass.
constexpr int kMaxSplits = 8;
constexpr int kMinTilesPerSplit = 8;   // >= 1024 keys per split: below that the prologue/epilogue of a CTA dominates

int choose_splits(int BH, int Nq, int nk, int dtype) {
  if (dtype != RINGX_BF16 || Nq % 256 || nk % 128) return 1;
  const long long ctas = (long long)BH * (Nq / 256);
  const int kSmCount = sm_count();       // of the current device: the same value sizes the workspace and picks the grid
  if (ctas >= 2 * kSmCount) return 1;
  const int tiles = nk / 128;
  auto eff = [kSmCount](long long n) { return (double)n / (double)(((n + kSmCount - 1) / kSmCount) * kSmCount); };
  int best = 1;
  double best_eff = eff(ctas);
  for (int s = 2; s <= kMaxSplits; ++s) {
    if (tiles % s || tiles / s < kMinTilesPerSplit) continue;
    const double e = eff(ctas * s) * (1.0 - 0.01 * s);     // every split costs one more partial to write and merge
    if (e > best_eff * 1.05) { best = s; best_eff = e; }
  }
  return best;
}

struct SplitScratch {
  int splits = 1;
  float* parts = nullptr;     // [splits][R,d]
  float* lses = nullptr;      // [splits][R]
  float* lse_tmp = nullptr;   // [R]: the merged lse when the caller's lse_out aliases lse_acc
  size_t bytes = 0;
};

SplitScratch carve_split(void* ws, size_t R, int d, int splits) {
  SplitScratch sp;
  sp.splits = splits;
  if (splits <= 1) return sp;
  char* p = static_cast<char*>(ws);
  size_t off = 0;
  auto take = [&](size_t n) {
    char* r = p ? p + off : nullptr;
    off += align_up(n);
    return r;
  };
  sp.parts = reinterpret_cast<float*>(take((size_t)splits * R * d * sizeof(float)));
  sp.lses = reinterpret_cast<float*>(take((size_t)splits * R * sizeof(float)));
  sp.lse_tmp = reinterpret_cast<float*>(take(R * sizeof(float)));
  sp.bytes = off;
  return sp;
}

struct FwdWorkspace {
  float* o_acc = nullptr;      // running (merged) output, fp32 [R,d]   (bf16 only; f32 uses `o` itself)
  float* lse_acc = nullptr;    // running LSE [R]                        (bf16 only; f32 uses `lse`)
  float* o_part = nullptr;     // loc_out of the current pass, fp32 [R,d]   (f32 only)
  float* lse_part = nullptr;   // loc_lse of the current pass [R]           (f32 only)
  SplitScratch split;          // split-KV scratch (splits == 1: none)
  size_t bytes = 0;
};

FwdWorkspace carve_fwd(void* ws, int B, int H, int N, int d, int kv_chunk, int dtype) {
  FwdWorkspace w;
  const size_t R = (size_t)B * H * N;
  char* p = static_cast<char*>(ws);
  size_t off = 0;
  auto take = [&](size_t n) {
    char* r = p ? p + off : nullptr;
    off += align_up(n);
    return r;
  };
  // (a ragged sequence or a short last chunk: no split-KV -- the passes would not all split alike)
  w.split = carve_split(nullptr, R, d, (N % 128 || N % kv_chunk) ? 1 : choose_splits(B * H, N, kv_chunk, dtype));
  if (w.split.splits > 1) w.split = carve_split(take(w.split.bytes), R, d, w.split.splits);
  if (kv_chunk >= N) {           // single pass: the chunk kernel writes (o, lse) directly
    w.bytes = off;
    return w;
  }
  if (dtype == RINGX_BF16) {   // the chunk kernel folds each pass into the running accumulator itself
    w.o_acc = reinterpret_cast<float*>(take(R * d * sizeof(float)));
    w.lse_acc = reinterpret_cast<float*>(take(R * sizeof(float)));
  } else {                     // fp32: partials of the current pass, merged by lse_merge into the caller's o/lse
    w.o_part = reinterpret_cast<float*>(take(R * d * sizeof(float)));
    w.lse_part = reinterpret_cast<float*>(take(R * sizeof(float)));
  }
  w.bytes = off;
  return w;
}

struct BwdWorkspace {
  float* D = nullptr;        // D_i = dO_i . O_i, [R]
  float* lse2 = nullptr;     // LSE_i * log2(e), [R]
  float* dq_acc = nullptr;   // fp32 dQ accumulator [R,d]
  float* dq_qs = nullptr;    // [R] per-row scales of the fixed-point dQ accumulator (deterministic mode)
  float* kvmax = nullptr;    // [2*B*H] scratch of launch_dq_fixed_scale
  size_t bytes = 0;
};

BwdWorkspace carve_bwd(void* ws, int B, int H, int N, int d) {
  BwdWorkspace w;
  const size_t R = (size_t)B * H * N;
  const size_t R_stat = (size_t)B * H * ((N + 127) / 128 * 128);   // D, lse2: every head padded to the 128-row tile
  char* p = static_cast<char*>(ws);
  w.D = reinterpret_cast<float*>(p);
  size_t off = align_up(R_stat * sizeof(float));
  w.lse2 = reinterpret_cast<float*>(p ? p + off : nullptr);
  off += align_up(R_stat * sizeof(float));
  w.dq_acc = reinterpret_cast<float*>(p ? p + off : nullptr);
  off += align_up(R * d * sizeof(float));
  w.dq_qs = reinterpret_cast<float*>(p ? p + off : nullptr);
  off += align_up(R * sizeof(float));
  w.kvmax = reinterpret_cast<float*>(p ? p + off : nullptr);
  off += align_up((size_t)B * H * 2 * sizeof(float));
  w.bytes = off;
  return w;
}

// process-wide, not per thread: a backward launched by an autograd worker thread must see the flag the user set on
// the main thread (torch runs `backward` of an autograd.Function on its own device thread)
std::atomic<int> g_deterministic{0};

// side stream + events of ringx_attn_fwd_bwd_host (host objects only; no device memory)
struct HostOverlap {
  int device = -1;
  cudaStream_t side = nullptr;
  std::vector<cudaEvent_t> events;
};
thread_local HostOverlap tl_overlap;

// side stream of the current device and at least n_events events (created on first use, then reused)
int overlap_prepare(HostOverlap& ov, int n_events) {
  cudaError_t ce;
  int dev = 0;
  if ((ce = cudaGetDevice(&dev)) != cudaSuccess) { cudaGetLastError(); return RINGX_ERR_CUDA; }
  if (!ov.side || ov.device != dev) {      // (objects of another device are abandoned, not reused)
    ov.device = dev;
    ov.events.clear();
    if ((ce = cudaStreamCreateWithFlags(&ov.side, cudaStreamNonBlocking)) != cudaSuccess) { cudaGetLastError(); return RINGX_ERR_CUDA; }
  }
  while ((int)ov.events.size() < n_events) {
    cudaEvent_t e;
    if ((ce = cudaEventCreateWithFlags(&e, cudaEventDisableTiming)) != cudaSuccess) { cudaGetLastError(); return RINGX_ERR_CUDA; }
    ov.events.push_back(e);
  }
  return RINGX_OK;
}

// Set by ringx_attn_fwd_bwd_host around its calls of the chunk loops: pass c of the forward waits for kv_ready[c] (the
// K,V rows of chunk c have arrived from the host); the backward records pass_done[c] after pass c (its dK,dV rows are final).
struct ChunkHooks {
  const cudaEvent_t* kv_ready = nullptr;
  const cudaEvent_t* pass_done = nullptr;
};
thread_local ChunkHooks tl_hooks;

// ---- optional live per-kernel timing (ringx_profile_*): CUDA events around each launch, per thread
struct Profile {
  bool on = false;
  std::vector<cudaEvent_t> pool;     // start/stop pairs, reused across reads
  std::vector<int> kinds;            // kind of pair i (events pool[2i], pool[2i+1])
};
thread_local Profile tl_prof;

struct Timed {   // RAII: brackets the launches made during its lifetime
  cudaStream_t stream;
  cudaEvent_t stop = nullptr;
  Timed(int kind, cudaStream_t s) : stream(s) {
    Profile& p = tl_prof;
    if (!p.on) return;
    const size_t i = p.kinds.size();
    while (p.pool.size() < 2 * (i + 1)) {
      cudaEvent_t e;
      if (cudaEventCreate(&e) != cudaSuccess) { cudaGetLastError(); return; }
      p.pool.push_back(e);
    }
    p.kinds.push_back(kind);
    cudaEventRecord(p.pool[2 * i], stream);
    stop = p.pool[2 * i + 1];
  }
  ~Timed() { if (stop) cudaEventRecord(stop, stream); }
};

int cuda_status(cudaError_t e) {
  if (e == cudaSuccess) return RINGX_OK;
  cudaGetLastError();
  return RINGX_ERR_CUDA;
}

}  // namespace

void count_launch(int n) { tl_launches += n; }

int sm_count() {
  static int cached[kMaxDevices];   // 0 = unknown (benign race: every writer stores the same value)
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) {
    cudaGetLastError();
    return 148;
  }
  if (dev >= 0 && dev < kMaxDevices && cached[dev]) return cached[dev];
  int n = 0;
  if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) {
    cudaGetLastError();
    return 148;
  }
  if (dev >= 0 && dev < kMaxDevices) cached[dev] = n;
  return n;
}

bool make_tmap_2d(CUtensorMap* out, const void* base, CUtensorMapDataType dt, int elem_bytes, uint64_t rows,
                  uint64_t cols, uint32_t box_rows, uint32_t box_cols, TmapSwizzle swz) {
  EncodeFn enc = encode_fn();
  if (!enc) return false;
  cuuint64_t dims[2] = {cols, rows};
  cuuint64_t strides[1] = {cols * (uint64_t)elem_bytes};
  cuuint32_t box[2] = {box_cols, box_rows};
  cuuint32_t es[2] = {1, 1};
  CUresult r = enc(out, dt, 2, const_cast<void*>(base), dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                   swz == kSwizzle128B ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_NONE,
                   CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS;
}

// 2-D view with a row pitch of `pitch_cols` elements (>= cols): columns >= cols are out of bounds (zero on load, skipped on
// store / reduce)
bool make_tmap_2d_pitched(CUtensorMap* out, const void* base, CUtensorMapDataType dt, int elem_bytes, uint64_t rows,
                          uint64_t cols, uint64_t pitch_cols, uint32_t box_rows, uint32_t box_cols, TmapSwizzle swz) {
  EncodeFn enc = encode_fn();
  if (!enc) return false;
  cuuint64_t dims[2] = {cols, rows};
  cuuint64_t strides[1] = {pitch_cols * (uint64_t)elem_bytes};
  cuuint32_t box[2] = {box_cols, box_rows};
  cuuint32_t es[2] = {1, 1};
  CUresult r = enc(out, dt, 2, const_cast<void*>(base), dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                   swz == kSwizzle128B ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_NONE,
                   CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS;
}

// 3-D view [heads][rows][cols] (row-major, contiguous), box = {box_cols, box_rows, 1}: a box that runs past the last row
// of a head is zero-filled on load and clipped on store / reduce (ragged sequence lengths)
bool make_tmap_3d(CUtensorMap* out, const void* base, CUtensorMapDataType dt, int elem_bytes, uint64_t heads, uint64_t rows,
                  uint64_t cols, uint32_t box_rows, uint32_t box_cols, TmapSwizzle swz) {
  EncodeFn enc = encode_fn();
  if (!enc) return false;
  cuuint64_t dims[3] = {cols, rows, heads};
  cuuint64_t strides[2] = {cols * (uint64_t)elem_bytes, rows * cols * (uint64_t)elem_bytes};
  cuuint32_t box[3] = {box_cols, box_rows, 1};
  cuuint32_t es[3] = {1, 1, 1};
  CUresult r = enc(out, dt, 3, const_cast<void*>(base), dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                   swz == kSwizzle128B ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_NONE,
                   CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS;
}

// One KV-chunk pass, either dtype.  `epilogue` (kernels.cuh, kFwdEpi*): partial / final / folded into (o_acc, lse_acc).
// The fp32 path has the partial epilogue only.
static cudaError_t chunk_pass(const void* q, const void* k, const void* v, void* o_out, float* lse_out,
                              const float* o_acc, const float* lse_acc, int BH, int Nq, int nk_stride, int k_off,
                              int nk, int d, float scale, int dtype, int epilogue, cudaStream_t stream,
                              const SplitScratch* sp = nullptr) {
  if (dtype == RINGX_F32) {
    Timed timed(RINGX_PROFILE_ATTN_FWD, stream);
    return launch_attn_chunk_f32(static_cast<const float*>(q), static_cast<const float*>(k),
                                 static_cast<const float*>(v), static_cast<float*>(o_out), lse_out, BH, Nq, nk_stride,
                                 k_off, nk, d, scale, stream);
  }
  if (!sp || sp->splits <= 1) {
    Timed timed(RINGX_PROFILE_ATTN_FWD, stream);
    return launch_attn_chunk_fwd_sm100(q, k, v, o_out, lse_out, o_acc, lse_acc, BH, Nq, nk_stride, k_off, nk, d, scale,
                                       epilogue, 1, stream);
  }
  // split-KV: gridDim.z splits of the keys write fp32 partials, one Eq. 5 kernel combines them (and the running
  // accumulator, for the fold epilogues) into what the unsplit pass would have produced
  cudaError_t e;
  {
    Timed timed(RINGX_PROFILE_ATTN_FWD, stream);
    e = launch_attn_chunk_fwd_sm100(q, k, v, sp->parts, sp->lses, nullptr, nullptr, BH, Nq, nk_stride, k_off, nk, d, scale,
                                    kFwdEpiPartial, sp->splits, stream);
  }
  if (e != cudaSuccess) return e;
  const bool fold = epilogue == kFwdEpiFold || epilogue == kFwdEpiFoldFinal;
  const bool out_bf16 = epilogue == kFwdEpiFinal || epilogue == kFwdEpiFoldFinal;
  const long long R = (long long)BH * Nq;
  float* lse_dst = (fold && lse_out == lse_acc) ? sp->lse_tmp : lse_out;   // other threads of a row still read lse_acc
  {
    Timed timed(RINGX_PROFILE_MERGE, stream);
    e = launch_split_merge(sp->parts, sp->lses, R, d, sp->splits, fold ? o_acc : nullptr, fold ? lse_acc : nullptr, o_out,
                           lse_dst, out_bf16 ? RINGX_BF16 : RINGX_F32, stream);
  }
  count_launch();
  if (e != cudaSuccess) return e;
  if (lse_dst != lse_out) e = cudaMemcpyAsync(lse_out, lse_dst, (size_t)R * sizeof(float), cudaMemcpyDeviceToDevice, stream);
  return e;
}

}  // namespace ringx

using namespace ringx;

extern "C" {

size_t ringx_attn_fwd_workspace_bytes(int B, int H, int N, int d, int kv_chunk, int dtype) {
  if (check_shape(B, H, N, d, kv_chunk, 1.f, dtype, false, true) != RINGX_OK) return 0;
  return carve_fwd(nullptr, B, H, N, d, kv_chunk, dtype).bytes;
}

size_t ringx_attn_bwd_workspace_bytes(int B, int H, int N, int d, int kv_chunk, int dtype) {
  if (check_shape(B, H, N, d, kv_chunk, 1.f, dtype, true, true) != RINGX_OK) return 0;
  return carve_bwd(nullptr, B, H, N, d).bytes;
}

size_t ringx_attn_fwd_host_workspace_bytes(int B, int H, int N, int d, int kv_chunk, int dtype) {
  if (check_shape(B, H, N, d, kv_chunk, 1.f, dtype, false, true) != RINGX_OK) return 0;
  const size_t e = dtype == RINGX_F32 ? 4 : 2;
  const size_t R = (size_t)B * H * N;
  return 4 * align_up(R * d * e) + align_up(R * sizeof(float)) + carve_fwd(nullptr, B, H, N, d, kv_chunk, dtype).bytes;
}

// Shared forward driver.  q,o: Nq rows per (batch, kv head); k,v: N rows per (batch, kv head); Nq = G*N with G query
// heads per kv head (G = 1: plain multi-head attention) -- the G heads that share a K,V head are adjacent in memory,
// so they are simply G*N query rows of one [BH, Nq, d] problem.
static int fwd_core(const void* q, const void* k, const void* v, void* o, float* lse, int BH, int Nq, int N, int d,
                    int kv_chunk, float scale, int dtype, const FwdWorkspace& w, cudaStream_t stream) {
  const long long R = (long long)BH * Nq;
  const int n_chunks = (N + kv_chunk - 1) / kv_chunk;      // the last chunk may be short (and its last key tile ragged)
  const int nk_last = N - (n_chunks - 1) * kv_chunk;
  if (n_chunks == 1) {
    cudaError_t e = chunk_pass(q, k, v, o, lse, nullptr, nullptr, BH, Nq, N, 0, N, d, scale, dtype, kFwdEpiFinal, stream,
                               &w.split);
    return e == cudaSuccess ? RINGX_OK : cuda_status(e);
  }
  for (int c = 0; c < n_chunks; ++c) {
    const bool first = c == 0, last = c == n_chunks - 1;
    if (tl_hooks.kv_ready && cudaStreamWaitEvent(stream, tl_hooks.kv_ready[c], 0) != cudaSuccess) return RINGX_ERR_CUDA;
    cudaError_t e;
    if (dtype == RINGX_BF16) {
      // Eq. 5, two operands, folded left to right in the chunk kernel's epilogue: the running (o_acc, lse_acc) stays
      // fp32 in the workspace; the last pass writes the caller's bf16 o and lse
      if (first)
        e = chunk_pass(q, k, v, w.o_acc, w.lse_acc, nullptr, nullptr, BH, Nq, N, 0, kv_chunk, d, scale, dtype,
                       kFwdEpiPartial, stream, &w.split);
      else if (!last)
        e = chunk_pass(q, k, v, w.o_acc, w.lse_acc, w.o_acc, w.lse_acc, BH, Nq, N, c * kv_chunk, kv_chunk, d, scale,
                       dtype, kFwdEpiFold, stream, &w.split);
      else
        e = chunk_pass(q, k, v, o, lse, w.o_acc, w.lse_acc, BH, Nq, N, c * kv_chunk, nk_last, d, scale, dtype,
                       kFwdEpiFoldFinal, stream, &w.split);
      if (e != cudaSuccess) return cuda_status(e);
      continue;
    }
    // fp32: partials, then ringx_lse_merge's kernel, accumulating straight into the caller's o/lse
    float* o_acc = static_cast<float*>(o);
    e = chunk_pass(q, k, v, first ? o_acc : w.o_part, first ? lse : w.lse_part, nullptr, nullptr, BH, Nq, N,
                   c * kv_chunk, kv_chunk, d, scale, dtype, kFwdEpiPartial, stream);
    if (e != cudaSuccess) return cuda_status(e);
    if (first) continue;
    Timed timed(RINGX_PROFILE_MERGE, stream);
    e = launch_lse_merge(o_acc, lse, w.o_part, w.lse_part, o_acc, lse, R, d, RINGX_F32, RINGX_F32, stream);
    count_launch();
    if (e != cudaSuccess) return cuda_status(e);
  }
  return RINGX_OK;
}

static int check_gqa(int Hq, int Hkv) {
  if (Hq <= 0 || Hkv <= 0 || Hq % Hkv) return RINGX_ERR_BAD_SHAPE;
  return RINGX_OK;
}

int ringx_attn_fwd_gqa(const void* q, const void* k, const void* v, void* o, float* lse, int B, int Hq, int Hkv, int N,
                       int d, int kv_chunk, float scale, int dtype, void* workspace, size_t workspace_bytes,
                       void* stream_) {
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  if (!q || !k || !v || !o || !lse) return RINGX_ERR_NULL_PTR;
  int st = check_gqa(Hq, Hkv);
  if (st == RINGX_OK) st = check_shape(B, Hq, N, d, kv_chunk, scale, dtype, false, true);
  if (st != RINGX_OK) return st;
  if (!aligned16(q) || !aligned16(k) || !aligned16(v) || !aligned16(o) || !aligned16(lse)) return RINGX_ERR_MISALIGNED;
  const FwdWorkspace need = carve_fwd(nullptr, B, Hq, N, d, kv_chunk, dtype);
  if (need.bytes) {
    if (!workspace) return RINGX_ERR_NULL_PTR;
    if (reinterpret_cast<uintptr_t>(workspace) % kAlign) return RINGX_ERR_MISALIGNED;
    if (workspace_bytes < need.bytes) return RINGX_ERR_WORKSPACE_TOO_SMALL;
  }
  if ((st = check_arch()) != RINGX_OK) return st;
  tl_launches = 0;
  const int G = Hq / Hkv;
  st = fwd_core(q, k, v, o, lse, B * Hkv, G * N, N, d, kv_chunk, scale, dtype,
                carve_fwd(workspace, B, Hq, N, d, kv_chunk, dtype), stream);
  if (st != RINGX_OK) return st;
  tl_last_launches = tl_launches;
  return RINGX_OK;
}

int ringx_attn_fwd(const void* q, const void* k, const void* v, void* o, float* lse, int B, int H, int N, int d,
                   int kv_chunk, float scale, int dtype, void* workspace, size_t workspace_bytes, void* stream_) {
  return ringx_attn_fwd_gqa(q, k, v, o, lse, B, H, H, N, d, kv_chunk, scale, dtype, workspace, workspace_bytes, stream_);
}

// ---- multi-head latent attention shapes (d_qk = 192, d_v = 128): the same chunk loop on the MLA kernel
size_t ringx_attn_fwd_mla_workspace_bytes(int B, int H, int N, int d_qk, int d_v, int kv_chunk) {
  if (d_qk != 192 || d_v != 128 || check_shape(B, H, N, d_v, kv_chunk, 1.f, RINGX_BF16, false, true) != RINGX_OK) return 0;
  if (kv_chunk >= N) return 0;
  const size_t R = (size_t)B * H * N;
  return align_up(R * d_v * sizeof(float)) + align_up(R * sizeof(float));
}

int ringx_attn_fwd_mla(const void* q, const void* k, const void* v, void* o, float* lse, int B, int H, int N, int d_qk,
                       int d_v, int kv_chunk, float scale, int dtype, void* workspace, size_t workspace_bytes,
                       void* stream_) {
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  if (!q || !k || !v || !o || !lse) return RINGX_ERR_NULL_PTR;
  if (dtype != RINGX_BF16) return RINGX_ERR_BAD_DTYPE;
  if (d_qk != 192 || d_v != 128) return RINGX_ERR_BAD_SHAPE;
  int st = check_shape(B, H, N, d_v, kv_chunk, scale, dtype, false, true);
  if (st != RINGX_OK) return st;
  if (!aligned16(q) || !aligned16(k) || !aligned16(v) || !aligned16(o) || !aligned16(lse)) return RINGX_ERR_MISALIGNED;
  const size_t need = ringx_attn_fwd_mla_workspace_bytes(B, H, N, d_qk, d_v, kv_chunk);
  if (need) {
    if (!workspace) return RINGX_ERR_NULL_PTR;
    if (reinterpret_cast<uintptr_t>(workspace) % kAlign) return RINGX_ERR_MISALIGNED;
    if (workspace_bytes < need) return RINGX_ERR_WORKSPACE_TOO_SMALL;
  }
  if ((st = check_arch()) != RINGX_OK) return st;
  tl_launches = 0;
  const int BH = B * H, n_chunks = (N + kv_chunk - 1) / kv_chunk;      // the last chunk may be short (ragged lengths)
  const size_t R = (size_t)BH * N;
  float* o_acc = static_cast<float*>(workspace);
  float* lse_acc = need ? reinterpret_cast<float*>(static_cast<char*>(workspace) + align_up(R * d_v * sizeof(float))) : nullptr;
  for (int c = 0; c < n_chunks; ++c) {
    const bool first = c == 0, last = c == n_chunks - 1;
    const int epi = n_chunks == 1 ? kFwdEpiFinal : first ? kFwdEpiPartial : last ? kFwdEpiFoldFinal : kFwdEpiFold;
    void* o_dst = (epi == kFwdEpiFinal || epi == kFwdEpiFoldFinal) ? o : static_cast<void*>(o_acc);
    float* l_dst = (epi == kFwdEpiFinal || epi == kFwdEpiFoldFinal) ? lse : lse_acc;
    cudaError_t e;
    {
      Timed timed(RINGX_PROFILE_ATTN_FWD, stream);
      e = launch_attn_chunk_fwd_mla_sm100(q, k, v, o_dst, l_dst, o_acc, lse_acc, BH, N, N, c * kv_chunk,
                                          last ? N - c * kv_chunk : kv_chunk, scale, epi, stream);
    }
    if (e != cudaSuccess) return cuda_status(e);
  }
  tl_last_launches = tl_launches;
  return RINGX_OK;
}

// backward of the same shapes: D / lse2 preprocess (d_v = 128 wide), one pass of the MLA backward kernel per KV chunk into
// the transposed fp32 dQ accumulator, transpose + bf16 cast of dQ
size_t ringx_attn_bwd_mla_workspace_bytes(int B, int H, int N, int d_qk, int d_v, int kv_chunk) {
  if (d_qk != 192 || d_v != 128 || check_shape(B, H, N, d_v, kv_chunk, 1.f, RINGX_BF16, true, true) != RINGX_OK) return 0;
  const size_t R = (size_t)B * H * N, Rp = (size_t)B * H * ((N + 127) / 128 * 128);    // Rp: every head padded to 128 rows
  // D, lse2 (padded), the transposed dQ accumulator (rows of padded length), and for deterministic mode the per-query
  // fixed-point scales + K/V maxima
  return 2 * align_up(Rp * sizeof(float)) + align_up(R * sizeof(float)) + align_up(Rp * d_qk * sizeof(float)) +
         align_up((size_t)B * H * 2 * sizeof(float));
}

int ringx_attn_bwd_mla(const void* q, const void* k, const void* v, const void* o, const float* lse, const void* dO,
                       void* dq, void* dk, void* dv, int B, int H, int N, int d_qk, int d_v, int kv_chunk, float scale,
                       int dtype, void* workspace, size_t workspace_bytes, void* stream_) {
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  if (!q || !k || !v || !o || !lse || !dO || !dq || !dk || !dv) return RINGX_ERR_NULL_PTR;
  if (dtype != RINGX_BF16) return RINGX_ERR_BAD_DTYPE;
  if (d_qk != 192 || d_v != 128) return RINGX_ERR_BAD_SHAPE;
  int st = check_shape(B, H, N, d_v, kv_chunk, scale, dtype, true, true);
  if (st != RINGX_OK) return st;
  if ((long long)B * H * d_qk > 0x7FFFFFFFLL) return RINGX_ERR_BAD_SHAPE;
  if (!aligned16(q) || !aligned16(k) || !aligned16(v) || !aligned16(o) || !aligned16(lse) || !aligned16(dO) ||
      !aligned16(dq) || !aligned16(dk) || !aligned16(dv))
    return RINGX_ERR_MISALIGNED;
  const size_t need = ringx_attn_bwd_mla_workspace_bytes(B, H, N, d_qk, d_v, kv_chunk);
  if (!workspace) return RINGX_ERR_NULL_PTR;
  if (reinterpret_cast<uintptr_t>(workspace) % kAlign) return RINGX_ERR_MISALIGNED;
  if (workspace_bytes < need) return RINGX_ERR_WORKSPACE_TOO_SMALL;
  if ((st = check_arch()) != RINGX_OK) return st;
  tl_launches = 0;
  const int BH = B * H;
  const size_t R = (size_t)BH * N, Rp = (size_t)BH * ((N + 127) / 128 * 128);
  float* D = static_cast<float*>(workspace);
  float* lse2 = reinterpret_cast<float*>(static_cast<char*>(workspace) + align_up(Rp * sizeof(float)));
  char* wp = static_cast<char*>(workspace) + 2 * align_up(Rp * sizeof(float));
  float* dq_acc_t = reinterpret_cast<float*>(wp);               // [BH*192][N rounded up to 128]
  wp += align_up(Rp * d_qk * sizeof(float));
  float* qs = reinterpret_cast<float*>(wp);
  float* kvmax = reinterpret_cast<float*>(wp + align_up(R * sizeof(float)));
  const bool fixed = g_deterministic.load(std::memory_order_relaxed) != 0;     // int32 fixed-point dQ (see bwd_core)
  cudaError_t e;
  {
    Timed timed(RINGX_PROFILE_BWD_AUX, stream);
    e = cudaMemsetAsync(dq_acc_t, 0, Rp * d_qk * sizeof(float), stream);
    if (e == cudaSuccess) e = launch_bwd_preprocess(o, dO, lse, D, lse2, nullptr, (long long)R, d_v, scale, false, stream, N);
    if (N % 128) count_launch();
    if (e == cudaSuccess && fixed) {
      e = launch_dq_fixed_scale(k, v, dO, D, kvmax, qs, BH, N, N, 0, N, d_qk, d_v, scale, stream);
      count_launch(2);
    }
  }
  count_launch();
  if (e != cudaSuccess) return cuda_status(e);
  const int n_chunks = (N + kv_chunk - 1) / kv_chunk;
  for (int c = 0; c < n_chunks; ++c) {
    Timed timed(RINGX_PROFILE_ATTN_BWD, stream);
    e = launch_attn_chunk_bwd_mla_sm100(q, k, v, dO, lse2, D, dq_acc_t, dk, dv, BH, N, N, c * kv_chunk,
                                        c + 1 < n_chunks ? kv_chunk : N - c * kv_chunk, scale,
                                        fixed ? qs : nullptr, RINGX_BF16, stream);
    if (e != cudaSuccess) return cuda_status(e);
  }
  {
    Timed timed(RINGX_PROFILE_BWD_AUX, stream);
    e = launch_dq_transpose_convert_mla(dq_acc_t, dq, BH, N, fixed ? qs : nullptr, stream);
  }
  count_launch();
  if (e != cudaSuccess) return cuda_status(e);
  tl_last_launches = tl_launches;
  return RINGX_OK;
}

// ---- the per-device RingX steps for the MLA widths (Nq != Nk; PAPER.md:137-147 with the layer design of PAPER.md:376)
static int check_mla_step(int B, int H, int Nq, int Nk, int d_qk, int d_v, float scale, int dtype, int nq_mult) {
  if (dtype != RINGX_BF16) return RINGX_ERR_BAD_DTYPE;
  if (d_qk != 192 || d_v != 128) return RINGX_ERR_BAD_SHAPE;
  if (B <= 0 || H <= 0 || Nq <= 0 || Nk <= 0 || Nk % 128 || Nq % nq_mult) return RINGX_ERR_BAD_SHAPE;
  if ((long long)B * H > 65535 || (long long)B * H * Nq > 0x7FFFFFFFLL || (long long)B * H * Nk > 0x7FFFFFFFLL)
    return RINGX_ERR_BAD_SHAPE;
  if (!(scale > 0.f) || !(scale < 3.0e38f)) return RINGX_ERR_BAD_SHAPE;
  return RINGX_OK;
}

int ringx_attn_chunk_fwd_mla(const void* q, const void* k, const void* v, const float* o_acc, const float* lse_acc,
                             void* o_out, float* lse_out, int B, int H, int Nq, int Nk, int d_qk, int d_v, float scale,
                             int dtype, int o_out_dtype, void* stream_) {
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  if (!q || !k || !v || !o_out || !lse_out || (o_acc == nullptr) != (lse_acc == nullptr)) return RINGX_ERR_NULL_PTR;
  if (o_out_dtype != RINGX_F32 && o_out_dtype != RINGX_BF16) return RINGX_ERR_BAD_DTYPE;
  int st = check_mla_step(B, H, Nq, Nk, d_qk, d_v, scale, dtype, 256);
  if (st != RINGX_OK) return st;
  if (!aligned16(q) || !aligned16(k) || !aligned16(v) || !aligned16(o_acc) || !aligned16(lse_acc) || !aligned16(o_out) ||
      !aligned16(lse_out))
    return RINGX_ERR_MISALIGNED;
  if (o_acc && o_out_dtype == RINGX_BF16 && (o_out == static_cast<const void*>(o_acc) || lse_out == lse_acc))
    return RINGX_ERR_BAD_SHAPE;              // a bf16 result cannot overwrite the fp32 accumulator
  if ((st = check_arch()) != RINGX_OK) return st;
  tl_launches = 0;
  const int epi = o_acc ? (o_out_dtype == RINGX_BF16 ? kFwdEpiFoldFinal : kFwdEpiFold)
                        : (o_out_dtype == RINGX_BF16 ? kFwdEpiFinal : kFwdEpiPartial);
  cudaError_t e;
  {
    Timed timed(RINGX_PROFILE_ATTN_FWD, stream);
    e = launch_attn_chunk_fwd_mla_sm100(q, k, v, o_out, lse_out, o_acc, lse_acc, B * H, Nq, Nk, 0, Nk, scale, epi, stream);
  }
  if (e != cudaSuccess) return cuda_status(e);
  tl_last_launches = tl_launches;
  return RINGX_OK;
}

size_t ringx_attn_bwd_partial_mla_workspace_bytes(int B, int H, int Nq) {
  if (B <= 0 || H <= 0 || Nq <= 0) return 0;
  return 2 * align_up((size_t)B * H * Nq * sizeof(float));
}

int ringx_attn_bwd_partial_mla(const void* q, const void* k, const void* v, const void* o, const float* lse,
                               const void* dO, float* dq_acc_t, void* dk, void* dv, int B, int H, int Nq, int Nk, int d_qk,
                               int d_v, float scale, int dtype, int dkv_dtype, int prepared, void* workspace,
                               size_t workspace_bytes, void* stream_) {
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  if (!q || !k || !v || !o || !lse || !dO || !dq_acc_t || !dk || !dv) return RINGX_ERR_NULL_PTR;
  if (dkv_dtype != RINGX_BF16 && dkv_dtype != RINGX_F32) return RINGX_ERR_BAD_DTYPE;
  int st = check_mla_step(B, H, Nq, Nk, d_qk, d_v, scale, dtype, 128);
  if (st != RINGX_OK) return st;
  if ((long long)B * H * d_qk > 0x7FFFFFFFLL) return RINGX_ERR_BAD_SHAPE;
  if (!aligned16(q) || !aligned16(k) || !aligned16(v) || !aligned16(o) || !aligned16(lse) || !aligned16(dO) ||
      !aligned16(dq_acc_t) || !aligned16(dk) || !aligned16(dv))
    return RINGX_ERR_MISALIGNED;
  const size_t need = ringx_attn_bwd_partial_mla_workspace_bytes(B, H, Nq);
  if (!workspace) return RINGX_ERR_NULL_PTR;
  if (reinterpret_cast<uintptr_t>(workspace) % kAlign) return RINGX_ERR_MISALIGNED;
  if (workspace_bytes < need) return RINGX_ERR_WORKSPACE_TOO_SMALL;
  if ((st = check_arch()) != RINGX_OK) return st;
  tl_launches = 0;
  const size_t R = (size_t)B * H * Nq;
  float* D = static_cast<float*>(workspace);
  float* lse2 = reinterpret_cast<float*>(static_cast<char*>(workspace) + align_up(R * sizeof(float)));
  cudaError_t e;
  if (!prepared) {
    {
      Timed timed(RINGX_PROFILE_BWD_AUX, stream);
      e = launch_bwd_preprocess(o, dO, lse, D, lse2, nullptr, (long long)R, d_v, scale, false, stream);
    }
    count_launch();
    if (e != cudaSuccess) return cuda_status(e);
  }
  {
    Timed timed(RINGX_PROFILE_ATTN_BWD, stream);
    e = launch_attn_chunk_bwd_mla_sm100(q, k, v, dO, lse2, D, dq_acc_t, dk, dv, B * H, Nq, Nk, 0, Nk, scale, nullptr, dkv_dtype,
                                        stream);
  }
  if (e != cudaSuccess) return cuda_status(e);
  tl_last_launches = tl_launches;
  return RINGX_OK;
}

int ringx_dq_finalize_mla(const float* dq_acc_t, void* dq, int B, int H, int Nq, int d_qk, void* stream_) {
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  if (!dq_acc_t || !dq) return RINGX_ERR_NULL_PTR;
  // Nq % 128 as ringx_attn_bwd_partial_mla, the only producer of dq_acc_t [B,H,d_qk,Nq]: the transpose reads it with a row
  // pitch of Nq rounded up to 128, which is the documented layout only when that is Nq itself
  if (d_qk != 192 || B <= 0 || H <= 0 || Nq <= 0 || Nq % 128 || (long long)B * H > 65535) return RINGX_ERR_BAD_SHAPE;
  if (!aligned16(dq_acc_t) || !aligned16(dq)) return RINGX_ERR_MISALIGNED;
  int st = check_arch();
  if (st != RINGX_OK) return st;
  tl_launches = 0;
  cudaError_t e;
  {
    Timed timed(RINGX_PROFILE_BWD_AUX, stream);
    e = launch_dq_transpose_convert_mla(dq_acc_t, dq, B * H, Nq, nullptr, stream);
  }
  count_launch();
  if (e != cudaSuccess) return cuda_status(e);
  tl_last_launches = tl_launches;
  return RINGX_OK;
}

int ringx_attn_chunk_fwd(const void* q, const void* k, const void* v, float* loc_out, float* loc_lse, int B, int H,
                         int Nq, int Nk, int d, float scale, int dtype, void* stream_) {
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  if (!q || !k || !v || !loc_out || !loc_lse) return RINGX_ERR_NULL_PTR;
  if (dtype != RINGX_F32 && dtype != RINGX_BF16) return RINGX_ERR_BAD_DTYPE;
  if (B <= 0 || H <= 0 || Nq <= 0 || Nk <= 0 || (d != 64 && d != 128)) return RINGX_ERR_BAD_SHAPE;
  if (dtype != RINGX_BF16 && (Nk % 128 || Nq % 128)) return RINGX_ERR_BAD_SHAPE;   // bf16: any Nq, Nk (ragged tiles)
  if ((long long)B * H > 65535 || (long long)B * H * Nq > 0x7FFFFFFFLL || (long long)B * H * Nk > 0x7FFFFFFFLL)
    return RINGX_ERR_BAD_SHAPE;
  if (!(scale > 0.f) || !(scale < 3.0e38f)) return RINGX_ERR_BAD_SHAPE;
  if (!aligned16(q) || !aligned16(k) || !aligned16(v) || !aligned16(loc_out) || !aligned16(loc_lse))
    return RINGX_ERR_MISALIGNED;
  int st = check_arch();
  if (st != RINGX_OK) return st;
  tl_launches = 0;
  cudaError_t e = chunk_pass(q, k, v, loc_out, loc_lse, nullptr, nullptr, B * H, Nq, Nk, 0, Nk, d, scale, dtype,
                             kFwdEpiPartial, stream);
  if (e != cudaSuccess) return cuda_status(e);
  tl_last_launches = tl_launches;
  return RINGX_OK;
}

int ringx_attn_chunk_fwd_fold(const void* q, const void* k, const void* v, float* o_acc, float* lse_acc, void* o_final,
                              float* lse_final, int B, int H, int Nq, int Nk, int d, float scale, int dtype,
                              void* stream_) {
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  if (!q || !k || !v || !o_acc || !lse_acc || (o_final == nullptr) != (lse_final == nullptr)) return RINGX_ERR_NULL_PTR;
  if (dtype != RINGX_BF16) return RINGX_ERR_BAD_DTYPE;
  if (B <= 0 || H <= 0 || Nq <= 0 || Nk <= 0 || (d != 64 && d != 128)) return RINGX_ERR_BAD_SHAPE;
  if ((long long)B * H > 65535 || (long long)B * H * Nq > 0x7FFFFFFFLL || (long long)B * H * Nk > 0x7FFFFFFFLL)
    return RINGX_ERR_BAD_SHAPE;
  if (!(scale > 0.f) || !(scale < 3.0e38f)) return RINGX_ERR_BAD_SHAPE;
  if (!aligned16(q) || !aligned16(k) || !aligned16(v) || !aligned16(o_acc) || !aligned16(lse_acc) ||
      !aligned16(o_final) || !aligned16(lse_final))
    return RINGX_ERR_MISALIGNED;
  int st = check_arch();
  if (st != RINGX_OK) return st;
  tl_launches = 0;
  cudaError_t e = o_final ? chunk_pass(q, k, v, o_final, lse_final, o_acc, lse_acc, B * H, Nq, Nk, 0, Nk, d, scale, dtype,
                                       kFwdEpiFoldFinal, stream)
                          : chunk_pass(q, k, v, o_acc, lse_acc, o_acc, lse_acc, B * H, Nq, Nk, 0, Nk, d, scale, dtype,
                                       kFwdEpiFold, stream);
  if (e != cudaSuccess) return cuda_status(e);
  tl_last_launches = tl_launches;
  return RINGX_OK;
}

size_t ringx_attn_chunk_fwd_ex_workspace_bytes(int B, int H, int Nq, int Nk, int d, int dtype) {
  if (B <= 0 || H <= 0 || Nq <= 0 || Nk <= 0 || (d != 64 && d != 128)) return 0;
  return carve_split(nullptr, (size_t)B * H * Nq, d, choose_splits(B * H, Nq, Nk, dtype)).bytes;
}

int ringx_attn_chunk_fwd_ex(const void* q, const void* k, const void* v, const float* o_acc, const float* lse_acc,
                            void* o_out, float* lse_out, int B, int H, int Nq, int Nk, int d, float scale, int dtype,
                            int o_out_dtype, void* workspace, size_t workspace_bytes, void* stream_) {
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  if (!q || !k || !v || !o_out || !lse_out || (o_acc == nullptr) != (lse_acc == nullptr)) return RINGX_ERR_NULL_PTR;
  if (dtype != RINGX_BF16) return RINGX_ERR_BAD_DTYPE;
  if (o_out_dtype != RINGX_F32 && o_out_dtype != RINGX_BF16) return RINGX_ERR_BAD_DTYPE;
  if (B <= 0 || H <= 0 || Nq <= 0 || Nk <= 0 || (d != 64 && d != 128)) return RINGX_ERR_BAD_SHAPE;
  if ((long long)B * H > 65535 || (long long)B * H * Nq > 0x7FFFFFFFLL || (long long)B * H * Nk > 0x7FFFFFFFLL)
    return RINGX_ERR_BAD_SHAPE;
  if (!(scale > 0.f) || !(scale < 3.0e38f)) return RINGX_ERR_BAD_SHAPE;
  if (!aligned16(q) || !aligned16(k) || !aligned16(v) || !aligned16(o_acc) || !aligned16(lse_acc) || !aligned16(o_out) ||
      !aligned16(lse_out))
    return RINGX_ERR_MISALIGNED;
  if (o_acc && o_out_dtype == RINGX_BF16 && (o_out == static_cast<const void*>(o_acc) || lse_out == lse_acc))
    return RINGX_ERR_BAD_SHAPE;              // a bf16 result cannot overwrite the fp32 accumulator
  const size_t need = ringx_attn_chunk_fwd_ex_workspace_bytes(B, H, Nq, Nk, d, dtype);
  if (need) {
    if (!workspace) return RINGX_ERR_NULL_PTR;
    if (reinterpret_cast<uintptr_t>(workspace) % kAlign) return RINGX_ERR_MISALIGNED;
    if (workspace_bytes < need) return RINGX_ERR_WORKSPACE_TOO_SMALL;
  }
  int st = check_arch();
  if (st != RINGX_OK) return st;
  tl_launches = 0;
  const SplitScratch sp = carve_split(workspace, (size_t)B * H * Nq, d, choose_splits(B * H, Nq, Nk, dtype));
  const int epi = o_acc ? (o_out_dtype == RINGX_BF16 ? kFwdEpiFoldFinal : kFwdEpiFold)
                        : (o_out_dtype == RINGX_BF16 ? kFwdEpiFinal : kFwdEpiPartial);
  cudaError_t e = chunk_pass(q, k, v, o_out, lse_out, o_acc, lse_acc, B * H, Nq, Nk, 0, Nk, d, scale, dtype, epi, stream, &sp);
  if (e != cudaSuccess) return cuda_status(e);
  tl_last_launches = tl_launches;
  return RINGX_OK;
}

int ringx_lse_merge(const void* o_a, const float* lse_a, const void* o_b, const float* lse_b, void* o_out,
                    float* lse_out, long long rows, int d, int o_in_dtype, int o_out_dtype, void* stream_) {
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  if (rows < 0 || d < 8 || d > 1024 || d % 8) return RINGX_ERR_BAD_SHAPE;
  if ((o_in_dtype != RINGX_F32 && o_in_dtype != RINGX_BF16) || (o_out_dtype != RINGX_F32 && o_out_dtype != RINGX_BF16))
    return RINGX_ERR_BAD_DTYPE;
  if (rows == 0) {
    tl_last_launches = 0;
    return RINGX_OK;
  }
  if (!o_a || !lse_a || !o_b || !lse_b || !o_out || !lse_out) return RINGX_ERR_NULL_PTR;
  if (!aligned16(o_a) || !aligned16(o_b) || !aligned16(o_out)) return RINGX_ERR_MISALIGNED;
  if ((reinterpret_cast<uintptr_t>(lse_a) | reinterpret_cast<uintptr_t>(lse_b) |
       reinterpret_cast<uintptr_t>(lse_out)) & 3u)
    return RINGX_ERR_MISALIGNED;
  tl_launches = 0;
  cudaError_t e;
  {
    Timed timed(RINGX_PROFILE_MERGE, stream);
    e = launch_lse_merge(o_a, lse_a, o_b, lse_b, o_out, lse_out, rows, d, o_in_dtype, o_out_dtype, stream);
  }
  count_launch();
  if (e != cudaSuccess) return cuda_status(e);
  tl_last_launches = tl_launches;
  return RINGX_OK;
}

// Shared backward driver: D/lse2 preprocess, one kernel pass per KV chunk of the nk keys, optional bf16 cast of dQ.
// q,o,dO,lse: Nq rows per head; k,v,dk,dv: Nk rows per head.  dq_acc fp32 [BH,Nq,d] (zeroed first when zero_dq).
// `prepared`: D and lse2 already hold this (o, lse, dO)'s values (an earlier step of the same RingX backward wrote them).
// dkv_dtype: dtype of dk, dv (bf16, or fp32 for one device's share of a cross-device sum).
// Deterministic mode (ringx_set_deterministic): det.qs != nullptr.  The passes accumulate dQ as int32 fixed point with
// the per-row scales det.qs (integer reduce-adds: order-independent) into det.fix -- dq_acc itself when the library owns
// the accumulator (dq_bf16 != nullptr), else a zeroed scratch that is added to the caller's fp32 dq_acc afterwards.
struct DetScratch {
  float* qs = nullptr;      // [BH*Nq]
  float* kvmax = nullptr;   // [2*BH]
  int* fix = nullptr;       // [BH*Nq*d] int32 (only when the caller owns dq_acc)
};

static int bwd_core(const void* q, const void* k, const void* v, const void* o, const float* lse, const void* dO,
                    float* D, float* lse2, float* dq_acc, bool zero_dq, void* dq_bf16, void* dk, void* dv, int BH,
                    int Nq, int Nk, int d, int kv_chunk, float scale, DetScratch det, cudaStream_t stream,
                    int dkv_dtype = RINGX_BF16, bool prepared = false) {
  const long long R = (long long)BH * Nq;
  cudaError_t e;
  const bool fixed = g_deterministic.load(std::memory_order_relaxed) != 0;
  if (fixed && (!det.qs || !det.kvmax || (!dq_bf16 && !det.fix))) return RINGX_ERR_WORKSPACE_TOO_SMALL;
  if (!prepared) {
    {
      Timed timed(RINGX_PROFILE_BWD_AUX, stream);
      e = launch_bwd_preprocess(o, dO, lse, D, lse2, dq_acc, R, d, scale, zero_dq, stream, Nq);
    }
    count_launch(Nq % 128 ? 2 : 1);
    if (e != cudaSuccess) return cuda_status(e);
  }
  float* pass_acc = dq_acc;
  if (fixed) {
    Timed timed(RINGX_PROFILE_BWD_AUX, stream);
    if (!dq_bf16) {
      pass_acc = reinterpret_cast<float*>(det.fix);
      if ((e = cudaMemsetAsync(det.fix, 0, (size_t)R * d * sizeof(int), stream)) != cudaSuccess) return cuda_status(e);
    }
    e = launch_dq_fixed_scale(k, v, dO, D, det.kvmax, det.qs, BH, Nq, Nk, 0, Nk, d, d, scale, stream);
    count_launch(2);
    if (e != cudaSuccess) return cuda_status(e);
  }
  const int n_chunks = (Nk + kv_chunk - 1) / kv_chunk;       // the last chunk may be short (and its last key tile ragged)
  for (int c = 0; c < n_chunks; ++c) {
    Timed timed(RINGX_PROFILE_ATTN_BWD, stream);
    const int nk_c = c + 1 < n_chunks ? kv_chunk : Nk - c * kv_chunk;
    e = launch_attn_chunk_bwd_sm100(q, k, v, dO, lse2, D, pass_acc, dk, dv, BH, Nq, Nk, c * kv_chunk, nk_c, d, scale,
                                    fixed ? det.qs : nullptr, dkv_dtype, stream);
    if (e != cudaSuccess) return cuda_status(e);
    if (tl_hooks.pass_done && (e = cudaEventRecord(tl_hooks.pass_done[c], stream)) != cudaSuccess) return cuda_status(e);
  }
  if (fixed) {
    Timed timed(RINGX_PROFILE_BWD_AUX, stream);
    e = launch_dq_fixed_finish(reinterpret_cast<const int*>(pass_acc), det.qs, dq_bf16, dq_acc, R, d, stream);
    count_launch();
    if (e != cudaSuccess) return cuda_status(e);
  } else if (dq_bf16) {
    Timed timed(RINGX_PROFILE_BWD_AUX, stream);
    e = launch_dq_convert(dq_acc, dq_bf16, R * d, 1.0f, stream);
    count_launch();
    if (e != cudaSuccess) return cuda_status(e);
  }
  return RINGX_OK;
}

int ringx_attn_bwd_gqa(const void* q, const void* k, const void* v, const void* o, const float* lse, const void* dO,
                       void* dq, void* dk, void* dv, int B, int Hq, int Hkv, int N, int d, int kv_chunk, float scale,
                       int dtype, void* workspace, size_t workspace_bytes, void* stream_) {
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  if (!q || !k || !v || !o || !lse || !dO || !dq || !dk || !dv) return RINGX_ERR_NULL_PTR;
  int st = check_gqa(Hq, Hkv);
  if (st == RINGX_OK) st = check_shape(B, Hq, N, d, kv_chunk, scale, dtype, true, true);
  if (st != RINGX_OK) return st;
  if (!aligned16(q) || !aligned16(k) || !aligned16(v) || !aligned16(o) || !aligned16(lse) || !aligned16(dO) ||
      !aligned16(dq) || !aligned16(dk) || !aligned16(dv))
    return RINGX_ERR_MISALIGNED;
  const BwdWorkspace need = carve_bwd(nullptr, B, Hq, N, d);
  if (!workspace) return RINGX_ERR_NULL_PTR;
  if (reinterpret_cast<uintptr_t>(workspace) % kAlign) return RINGX_ERR_MISALIGNED;
  if (workspace_bytes < need.bytes) return RINGX_ERR_WORKSPACE_TOO_SMALL;
  if ((st = check_arch()) != RINGX_OK) return st;

  tl_launches = 0;
  const BwdWorkspace w = carve_bwd(workspace, B, Hq, N, d);
  // the G = Hq/Hkv query heads of a kv head are G*N adjacent query rows: the CTA that owns a key tile walks all of them,
  // so dK, dV of the kv head are still written once, atomic-free
  const int G = Hq / Hkv;
  DetScratch det;
  det.qs = w.dq_qs;
  det.kvmax = w.kvmax;
  st = bwd_core(q, k, v, o, lse, dO, w.D, w.lse2, w.dq_acc, true, dq, dk, dv, B * Hkv, G * N, N, d, kv_chunk, scale,
                det, stream);
  if (st != RINGX_OK) return st;
  tl_last_launches = tl_launches;
  return RINGX_OK;
}

int ringx_attn_bwd(const void* q, const void* k, const void* v, const void* o, const float* lse, const void* dO,
                   void* dq, void* dk, void* dv, int B, int H, int N, int d, int kv_chunk, float scale, int dtype,
                   void* workspace, size_t workspace_bytes, void* stream_) {
  return ringx_attn_bwd_gqa(q, k, v, o, lse, dO, dq, dk, dv, B, H, H, N, d, kv_chunk, scale, dtype, workspace,
                            workspace_bytes, stream_);
}

size_t ringx_attn_bwd_partial_workspace_bytes(int B, int H, int Nq, int d) {
  if (B <= 0 || H <= 0 || Nq <= 0 || (d != 64 && d != 128)) return 0;
  const size_t R = (size_t)B * H * Nq;
  size_t bytes = 2 * align_up((size_t)B * H * ((Nq + 127) / 128 * 128) * sizeof(float));   // D, lse2: heads padded to 128 rows
  // deterministic mode: per-row scales, the K/V maxima and an int32 fixed-point image of this step's dQ contribution
  if (g_deterministic.load(std::memory_order_relaxed))
    bytes += align_up(R * sizeof(float)) + align_up((size_t)B * H * 2 * sizeof(float)) + align_up(R * d * sizeof(int));
  return bytes;
}

int ringx_attn_bwd_partial_ex(const void* q, const void* k, const void* v, const void* o, const float* lse,
                              const void* dO, float* dq_acc, void* dk, void* dv, int B, int H, int Nq, int Nk, int d,
                              float scale, int dtype, int dkv_dtype, int prepared, void* workspace,
                              size_t workspace_bytes, void* stream_) {
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  if (!q || !k || !v || !o || !lse || !dO || !dq_acc || !dk || !dv) return RINGX_ERR_NULL_PTR;
  if (dtype != RINGX_BF16) return RINGX_ERR_BAD_DTYPE;
  if (dkv_dtype != RINGX_BF16 && dkv_dtype != RINGX_F32) return RINGX_ERR_BAD_DTYPE;
  if (B <= 0 || H <= 0 || Nq <= 0 || Nk <= 0 || (d != 64 && d != 128)) return RINGX_ERR_BAD_SHAPE;
  if ((long long)B * H > 65535 || (long long)B * H * Nq > 0x7FFFFFFFLL || (long long)B * H * Nk > 0x7FFFFFFFLL)
    return RINGX_ERR_BAD_SHAPE;
  if (!(scale > 0.f) || !(scale < 3.0e38f)) return RINGX_ERR_BAD_SHAPE;
  if (!aligned16(q) || !aligned16(k) || !aligned16(v) || !aligned16(o) || !aligned16(lse) || !aligned16(dO) ||
      !aligned16(dq_acc) || !aligned16(dk) || !aligned16(dv))
    return RINGX_ERR_MISALIGNED;
  const size_t need = ringx_attn_bwd_partial_workspace_bytes(B, H, Nq, d);
  if (!workspace) return RINGX_ERR_NULL_PTR;
  if (reinterpret_cast<uintptr_t>(workspace) % kAlign) return RINGX_ERR_MISALIGNED;
  if (workspace_bytes < need) return RINGX_ERR_WORKSPACE_TOO_SMALL;
  int st = check_arch();
  if (st != RINGX_OK) return st;
  tl_launches = 0;
  float* D = static_cast<float*>(workspace);
  const size_t rb = align_up((size_t)B * H * ((Nq + 127) / 128 * 128) * sizeof(float));
  float* lse2 = reinterpret_cast<float*>(static_cast<char*>(workspace) + rb);
  DetScratch det;
  if (need > 2 * rb) {      // the workspace was sized in deterministic mode
    char* p = static_cast<char*>(workspace) + 2 * rb;
    const size_t qb = align_up((size_t)B * H * Nq * sizeof(float));
    det.qs = reinterpret_cast<float*>(p);
    det.kvmax = reinterpret_cast<float*>(p + qb);
    det.fix = reinterpret_cast<int*>(p + qb + align_up((size_t)B * H * 2 * sizeof(float)));
  }
  st = bwd_core(q, k, v, o, lse, dO, D, lse2, dq_acc, false, nullptr, dk, dv, B * H, Nq, Nk, d, Nk, scale, det, stream,
                dkv_dtype, prepared != 0);
  if (st != RINGX_OK) return st;
  tl_last_launches = tl_launches;
  return RINGX_OK;
}

int ringx_attn_bwd_partial(const void* q, const void* k, const void* v, const void* o, const float* lse,
                           const void* dO, float* dq_acc, void* dk, void* dv, int B, int H, int Nq, int Nk, int d,
                           float scale, int dtype, void* workspace, size_t workspace_bytes, void* stream_) {
  return ringx_attn_bwd_partial_ex(q, k, v, o, lse, dO, dq_acc, dk, dv, B, H, Nq, Nk, d, scale, dtype, RINGX_BF16, 0,
                                   workspace, workspace_bytes, stream_);
}

int ringx_dq_finalize(const float* dq_acc, void* dq, long long n, void* stream_) {
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  if (n < 0 || n % 4) return RINGX_ERR_BAD_SHAPE;
  if (n == 0) { tl_last_launches = 0; return RINGX_OK; }
  if (!dq_acc || !dq) return RINGX_ERR_NULL_PTR;
  if (!aligned16(dq_acc) || (reinterpret_cast<uintptr_t>(dq) & 7u)) return RINGX_ERR_MISALIGNED;
  tl_launches = 0;
  cudaError_t e;
  {
    Timed timed(RINGX_PROFILE_BWD_AUX, stream);
    e = launch_dq_convert(dq_acc, dq, n, 1.0f, stream);
  }
  count_launch();
  if (e != cudaSuccess) return cuda_status(e);
  tl_last_launches = tl_launches;
  return RINGX_OK;
}

static int check_eq5(const void* a, const void* b, const void* c, const void* d_, const void* e, long long rows, int d) {
  if (rows < 0 || d < 8 || d > 1024 || d % 8) return RINGX_ERR_BAD_SHAPE;
  if (rows == 0) return RINGX_OK;
  if (!a || !b || !c || !d_ || !e) return RINGX_ERR_NULL_PTR;
  return RINGX_OK;
}

int ringx_eq5_scale(const float* loc_out, const float* loc_lse, const float* lse_max, float* num, float* den,
                    long long rows, int d, void* stream_) {
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  int st = check_eq5(loc_out, loc_lse, lse_max, num, den, rows, d);
  if (st != RINGX_OK) return st;
  if (rows == 0) { tl_last_launches = 0; return RINGX_OK; }
  if (!aligned16(loc_out) || !aligned16(num)) return RINGX_ERR_MISALIGNED;
  tl_launches = 0;
  cudaError_t e;
  {
    Timed timed(RINGX_PROFILE_MERGE, stream);
    e = launch_eq5_scale(loc_out, loc_lse, lse_max, num, den, rows, d, stream);
  }
  count_launch();
  if (e != cudaSuccess) return cuda_status(e);
  tl_last_launches = tl_launches;
  return RINGX_OK;
}

int ringx_eq5_finalize(const float* num, const float* den, const float* lse_max, void* o_out, float* lse_out,
                       long long rows, int d, int o_out_dtype, void* stream_) {
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  if (o_out_dtype != RINGX_F32 && o_out_dtype != RINGX_BF16) return RINGX_ERR_BAD_DTYPE;
  int st = check_eq5(num, den, lse_max, o_out, lse_out, rows, d);
  if (st != RINGX_OK) return st;
  if (rows == 0) { tl_last_launches = 0; return RINGX_OK; }
  if (!aligned16(num) || !aligned16(o_out)) return RINGX_ERR_MISALIGNED;
  tl_launches = 0;
  cudaError_t e;
  {
    Timed timed(RINGX_PROFILE_MERGE, stream);
    e = launch_eq5_finalize(num, den, lse_max, o_out, lse_out, rows, d, o_out_dtype, stream);
  }
  count_launch();
  if (e != cudaSuccess) return cuda_status(e);
  tl_last_launches = tl_launches;
  return RINGX_OK;
}

int ringx_attn_fwd_host(const void* q_host, const void* k_host, const void* v_host, void* o_host, float* lse_host,
                        int B, int H, int N, int d, int kv_chunk, float scale, int dtype, void* workspace,
                        size_t workspace_bytes, void* stream_) {
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  if (!q_host || !k_host || !v_host || !o_host || !lse_host) return RINGX_ERR_NULL_PTR;
  int st = check_shape(B, H, N, d, kv_chunk, scale, dtype, false, true);
  if (st != RINGX_OK) return st;
  const size_t need = ringx_attn_fwd_host_workspace_bytes(B, H, N, d, kv_chunk, dtype);
  if (!workspace) return RINGX_ERR_NULL_PTR;
  if (reinterpret_cast<uintptr_t>(workspace) % kAlign) return RINGX_ERR_MISALIGNED;
  if (workspace_bytes < need) return RINGX_ERR_WORKSPACE_TOO_SMALL;
  const size_t e = dtype == RINGX_F32 ? 4 : 2;
  const size_t R = (size_t)B * H * N;
  const size_t tb = R * d * e, tba = align_up(tb);
  char* p = static_cast<char*>(workspace);
  void *dq = p, *dk = p + tba, *dv = p + 2 * tba, *dob = p + 3 * tba;
  float* dlse = reinterpret_cast<float*>(p + 4 * tba);
  char* inner = p + 4 * tba + align_up(R * sizeof(float));
  const size_t inner_bytes = workspace_bytes - (size_t)(inner - p);
  // q and the K,V rows of chunk c go up on a side stream in the order the passes need them (pass c waits for chunk c
  // only), so all but the first chunk's transfer is hidden behind the kernels.
  cudaError_t ce;
  const int n_chunks = (N + kv_chunk - 1) / kv_chunk;      // the last chunk may be short (ragged lengths)
  const bool pipelined = n_chunks >= 2 && n_chunks <= 64;
  if (pipelined) {
    HostOverlap& ov = tl_overlap;
    if ((st = overlap_prepare(ov, 3 + 2 * n_chunks)) != RINGX_OK) return st;
    cudaEvent_t* kv_ready = ov.events.data() + 3;
    const size_t head_pitch = (size_t)N * d * e, chunk_bytes = (size_t)kv_chunk * d * e;
    if ((ce = cudaEventRecord(ov.events[2], stream)) != cudaSuccess) return cuda_status(ce);
    if ((ce = cudaStreamWaitEvent(ov.side, ov.events[2], 0)) != cudaSuccess) return cuda_status(ce);
    if ((ce = cudaMemcpyAsync(dq, q_host, tb, cudaMemcpyHostToDevice, ov.side)) != cudaSuccess) return cuda_status(ce);
    for (int c = 0; c < n_chunks; ++c) {
      const size_t off = (size_t)c * chunk_bytes, this_bytes = c + 1 < n_chunks ? chunk_bytes : head_pitch - off;
      for (int w = 0; w < 2; ++w)
        if ((ce = cudaMemcpy2DAsync(static_cast<char*>(w == 0 ? dk : dv) + off, head_pitch,
                                    static_cast<const char*>(w == 0 ? k_host : v_host) + off, head_pitch, this_bytes,
                                    (size_t)B * H, cudaMemcpyHostToDevice, ov.side)) != cudaSuccess)
          return cuda_status(ce);
      if ((ce = cudaEventRecord(kv_ready[c], ov.side)) != cudaSuccess) return cuda_status(ce);
    }
    tl_hooks.kv_ready = kv_ready;
  } else {
    if ((ce = cudaMemcpyAsync(dq, q_host, tb, cudaMemcpyHostToDevice, stream)) != cudaSuccess) return cuda_status(ce);
    if ((ce = cudaMemcpyAsync(dk, k_host, tb, cudaMemcpyHostToDevice, stream)) != cudaSuccess) return cuda_status(ce);
    if ((ce = cudaMemcpyAsync(dv, v_host, tb, cudaMemcpyHostToDevice, stream)) != cudaSuccess) return cuda_status(ce);
  }
  st = ringx_attn_fwd(dq, dk, dv, dob, dlse, B, H, N, d, kv_chunk, scale, dtype, inner, inner_bytes, stream_);
  tl_hooks.kv_ready = nullptr;
  if (st != RINGX_OK) return st;
  if ((ce = cudaMemcpyAsync(o_host, dob, tb, cudaMemcpyDeviceToHost, stream)) != cudaSuccess) return cuda_status(ce);
  if ((ce = cudaMemcpyAsync(lse_host, dlse, R * sizeof(float), cudaMemcpyDeviceToHost, stream)) != cudaSuccess)
    return cuda_status(ce);
  if ((ce = cudaStreamSynchronize(stream)) != cudaSuccess) return cuda_status(ce);
  return RINGX_OK;
}

size_t ringx_attn_fwd_bwd_host_workspace_bytes(int B, int H, int N, int d, int kv_chunk, int dtype) {
  if (check_shape(B, H, N, d, kv_chunk, 1.f, dtype, true, true) != RINGX_OK ||
      check_shape(B, H, N, d, kv_chunk, 1.f, dtype, false, true) != RINGX_OK)
    return 0;
  const size_t R = (size_t)B * H * N;
  const size_t fw = carve_fwd(nullptr, B, H, N, d, kv_chunk, dtype).bytes, bw = carve_bwd(nullptr, B, H, N, d).bytes;
  return 8 * align_up(R * d * 2) + align_up(R * sizeof(float)) + (fw > bw ? fw : bw);
}

int ringx_attn_fwd_bwd_host(const void* q_host, const void* k_host, const void* v_host, const void* dO_host,
                            void* o_host, float* lse_host, void* dq_host, void* dk_host, void* dv_host, int B, int H,
                            int N, int d, int kv_chunk, float scale, int dtype, void* workspace,
                            size_t workspace_bytes, void* stream_) {
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  if (!q_host || !k_host || !v_host || !dO_host || !o_host || !lse_host || !dq_host || !dk_host || !dv_host)
    return RINGX_ERR_NULL_PTR;
  int st = check_shape(B, H, N, d, kv_chunk, scale, dtype, true, true);
  if (st == RINGX_OK) st = check_shape(B, H, N, d, kv_chunk, scale, dtype, false, true);
  if (st != RINGX_OK) return st;
  const size_t need = ringx_attn_fwd_bwd_host_workspace_bytes(B, H, N, d, kv_chunk, dtype);
  if (!workspace) return RINGX_ERR_NULL_PTR;
  if (reinterpret_cast<uintptr_t>(workspace) % kAlign) return RINGX_ERR_MISALIGNED;
  if (workspace_bytes < need) return RINGX_ERR_WORKSPACE_TOO_SMALL;
  const size_t R = (size_t)B * H * N;
  const size_t tb = R * d * 2, tba = align_up(tb);
  char* p = static_cast<char*>(workspace);
  void* t[8];   // q k v dO | o dq dk dv
  for (int i = 0; i < 8; ++i) t[i] = p + i * tba;
  float* dlse = reinterpret_cast<float*>(p + 8 * tba);
  char* inner = p + 8 * tba + align_up(R * sizeof(float));
  const size_t inner_bytes = workspace_bytes - (size_t)(inner - p);
  // Copies run on a side stream (host objects, created once per thread) so that they overlap the kernels: q and the
  // K,V rows of chunk c go up in the order the passes need them (pass c waits for chunk c only), dO goes up while the
  // forward runs, o and lse come down while the backward runs, and the dK,dV rows of chunk c -- final after pass c --
  // come down while the later passes run.  Only dq is copied after the last kernel.
  HostOverlap& ov = tl_overlap;
  cudaError_t ce;
  const int n_chunks = (N + kv_chunk - 1) / kv_chunk;      // the last chunk may be short (ragged lengths)
  const bool pipelined = n_chunks >= 2 && n_chunks <= 64;
  if ((st = overlap_prepare(ov, 3 + (pipelined ? 2 * n_chunks : 0))) != RINGX_OK) return st;
  cudaEvent_t ev_do_up = ov.events[0], ev_fwd_done = ov.events[1], ev_down = ov.events[2];
  cudaEvent_t* kv_ready = ov.events.data() + 3;
  cudaEvent_t* pass_done = kv_ready + n_chunks;
  const int BH = B * H;
  const size_t row_bytes = (size_t)d * 2, head_pitch = (size_t)N * row_bytes, chunk_bytes = (size_t)kv_chunk * row_bytes;
  auto up = [&](void* dst, const void* src_, size_t bytes) {
    return cudaMemcpyAsync(dst, src_, bytes, cudaMemcpyHostToDevice, ov.side);
  };
  // ---- host -> device
  if ((ce = cudaEventRecord(ev_down, stream)) != cudaSuccess) return cuda_status(ce);          // order behind the caller's
  if ((ce = cudaStreamWaitEvent(ov.side, ev_down, 0)) != cudaSuccess) return cuda_status(ce);  // earlier work on `stream`
  if ((ce = up(t[0], q_host, tb)) != cudaSuccess) return cuda_status(ce);
  if (pipelined) {
    for (int c = 0; c < n_chunks; ++c) {
      const size_t off = (size_t)c * chunk_bytes, this_bytes = c + 1 < n_chunks ? chunk_bytes : head_pitch - off;
      for (int w = 1; w <= 2; ++w) {
        const char* src_ = static_cast<const char*>(w == 1 ? k_host : v_host) + off;
        if ((ce = cudaMemcpy2DAsync(static_cast<char*>(t[w]) + off, head_pitch, src_, head_pitch, this_bytes, BH,
                                    cudaMemcpyHostToDevice, ov.side)) != cudaSuccess)
          return cuda_status(ce);
      }
      if ((ce = cudaEventRecord(kv_ready[c], ov.side)) != cudaSuccess) return cuda_status(ce);
    }
  } else {
    if ((ce = up(t[1], k_host, tb)) != cudaSuccess || (ce = up(t[2], v_host, tb)) != cudaSuccess) return cuda_status(ce);
    if ((ce = cudaEventRecord(ev_fwd_done, ov.side)) != cudaSuccess) return cuda_status(ce);
    if ((ce = cudaStreamWaitEvent(stream, ev_fwd_done, 0)) != cudaSuccess) return cuda_status(ce);
  }
  if ((ce = up(t[3], dO_host, tb)) != cudaSuccess) return cuda_status(ce);
  if ((ce = cudaEventRecord(ev_do_up, ov.side)) != cudaSuccess) return cuda_status(ce);
  // ---- forward
  if (pipelined) tl_hooks.kv_ready = kv_ready;
  st = ringx_attn_fwd(t[0], t[1], t[2], t[4], dlse, B, H, N, d, kv_chunk, scale, dtype, inner, inner_bytes, stream_);
  tl_hooks.kv_ready = nullptr;
  if (st != RINGX_OK) return st;
  const int fwd_launches = tl_last_launches;
  if ((ce = cudaEventRecord(ev_fwd_done, stream)) != cudaSuccess) return cuda_status(ce);
  if ((ce = cudaStreamWaitEvent(ov.side, ev_fwd_done, 0)) != cudaSuccess) return cuda_status(ce);
  if ((ce = cudaMemcpyAsync(o_host, t[4], tb, cudaMemcpyDeviceToHost, ov.side)) != cudaSuccess) return cuda_status(ce);
  if ((ce = cudaMemcpyAsync(lse_host, dlse, R * sizeof(float), cudaMemcpyDeviceToHost, ov.side)) != cudaSuccess)
    return cuda_status(ce);
  // ---- backward
  if ((ce = cudaStreamWaitEvent(stream, ev_do_up, 0)) != cudaSuccess) return cuda_status(ce);
  if (pipelined) tl_hooks.pass_done = pass_done;
  st = ringx_attn_bwd(t[0], t[1], t[2], t[4], dlse, t[3], t[5], t[6], t[7], B, H, N, d, kv_chunk, scale, dtype, inner,
                      inner_bytes, stream_);
  tl_hooks.pass_done = nullptr;
  if (st != RINGX_OK) return st;
  tl_last_launches += fwd_launches;
  // ---- device -> host (the waits are enqueued after the records they refer to)
  if (pipelined) {
    for (int c = 0; c < n_chunks; ++c) {
      const size_t off = (size_t)c * chunk_bytes, this_bytes = c + 1 < n_chunks ? chunk_bytes : head_pitch - off;
      if ((ce = cudaStreamWaitEvent(ov.side, pass_done[c], 0)) != cudaSuccess) return cuda_status(ce);
      for (int w = 0; w < 2; ++w) {
        char* dst_ = static_cast<char*>(w == 0 ? dk_host : dv_host) + off;
        if ((ce = cudaMemcpy2DAsync(dst_, head_pitch, static_cast<const char*>(t[6 + w]) + off, head_pitch, this_bytes,
                                    BH, cudaMemcpyDeviceToHost, ov.side)) != cudaSuccess)
          return cuda_status(ce);
      }
    }
  } else {
    if ((ce = cudaMemcpyAsync(dk_host, t[6], tb, cudaMemcpyDeviceToHost, stream)) != cudaSuccess ||
        (ce = cudaMemcpyAsync(dv_host, t[7], tb, cudaMemcpyDeviceToHost, stream)) != cudaSuccess)
      return cuda_status(ce);
  }
  if ((ce = cudaMemcpyAsync(dq_host, t[5], tb, cudaMemcpyDeviceToHost, stream)) != cudaSuccess) return cuda_status(ce);
  if ((ce = cudaEventRecord(ev_down, ov.side)) != cudaSuccess) return cuda_status(ce);
  if ((ce = cudaStreamWaitEvent(stream, ev_down, 0)) != cudaSuccess) return cuda_status(ce);
  if ((ce = cudaStreamSynchronize(stream)) != cudaSuccess) return cuda_status(ce);
  return RINGX_OK;
}

// ---- backward of the projections and of the block (derivative of Table II's GEMMs)
static int check_proj(int B, int S, int H, int d);
static int check_proj_bwd(int B, int S, int H, int d) {
  int st = check_proj(B, S, H, d);
  if (st != RINGX_OK) return st;
  if ((H * d) % 256) return RINGX_ERR_BAD_SHAPE;      // the MN-major operand tiles are not ragged
  return RINGX_OK;
}

int ringx_out_proj_bwd(const void* dy, const void* o, const void* w_o, void* d_o, float* dw_o, int B, int S, int H, int d,
                       void* stream_) {
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  int st = check_proj_bwd(B, S, H, d);
  if (st != RINGX_OK) return st;
  if (!dy || !o || !w_o || !d_o || !dw_o) return RINGX_ERR_NULL_PTR;
  if (!aligned16(dy) || !aligned16(o) || !aligned16(w_o) || !aligned16(d_o) || !aligned16(dw_o)) return RINGX_ERR_MISALIGNED;
  if ((st = check_arch()) != RINGX_OK) return st;
  tl_launches = 0;
  const size_t h = (size_t)H * d;
  cudaError_t e = cudaMemsetAsync(dw_o, 0, h * h * sizeof(float), stream);
  if (e != cudaSuccess) return cuda_status(e);
  {
    Timed timed(RINGX_PROFILE_PROJ, stream);
    e = launch_out_proj_bwd(dy, o, w_o, d_o, dw_o, B, S, H, d, stream);
  }
  if (e != cudaSuccess) return cuda_status(e);
  tl_last_launches = tl_launches;
  return RINGX_OK;
}

int ringx_qkv_proj_bwd(const void* dq, const void* dk, const void* dv, const void* x, const void* w_qkv, void* dx,
                       float* dw_qkv, int B, int S, int H, int d, void* stream_) {
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  int st = check_proj_bwd(B, S, H, d);
  if (st != RINGX_OK) return st;
  if (!dq || !dk || !dv || !x || !w_qkv || !dx || !dw_qkv) return RINGX_ERR_NULL_PTR;
  if (!aligned16(dq) || !aligned16(dk) || !aligned16(dv) || !aligned16(x) || !aligned16(w_qkv) || !aligned16(dx) ||
      !aligned16(dw_qkv))
    return RINGX_ERR_MISALIGNED;
  if ((st = check_arch()) != RINGX_OK) return st;
  tl_launches = 0;
  const size_t h = (size_t)H * d;
  cudaError_t e = cudaMemsetAsync(dw_qkv, 0, 3 * h * h * sizeof(float), stream);
  if (e != cudaSuccess) return cuda_status(e);
  {
    Timed timed(RINGX_PROFILE_PROJ, stream);
    e = launch_qkv_proj_bwd(dq, dk, dv, x, w_qkv, dx, dw_qkv, B, S, H, d, stream);
  }
  if (e != cudaSuccess) return cuda_status(e);
  tl_last_launches = tl_launches;
  return RINGX_OK;
}

size_t ringx_attn_block_bwd_workspace_bytes(int B, int S, int H, int d, int kv_chunk) {
  if (check_proj_bwd(B, S, H, d) != RINGX_OK) return 0;
  const size_t R = (size_t)B * H * S;
  return 4 * align_up(R * d * 2) + align_up(ringx_attn_bwd_workspace_bytes(B, H, S, d, kv_chunk, RINGX_BF16));
}

int ringx_attn_block_bwd(const void* x, const void* w_qkv, const void* w_o, const void* dy, const void* fwd_workspace,
                         void* dx, float* dw_qkv, float* dw_o, int B, int S, int H, int d, int kv_chunk, float scale,
                         void* workspace, size_t workspace_bytes, void* stream_) {
  int st = check_proj_bwd(B, S, H, d);
  if (st == RINGX_OK) st = check_shape(B, H, S, d, kv_chunk, scale, RINGX_BF16, true);
  if (st != RINGX_OK) return st;
  if (!x || !w_qkv || !w_o || !dy || !fwd_workspace || !dx || !dw_qkv || !dw_o || !workspace) return RINGX_ERR_NULL_PTR;
  if (reinterpret_cast<uintptr_t>(workspace) % kAlign || reinterpret_cast<uintptr_t>(fwd_workspace) % kAlign)
    return RINGX_ERR_MISALIGNED;
  if (workspace_bytes < ringx_attn_block_bwd_workspace_bytes(B, S, H, d, kv_chunk)) return RINGX_ERR_WORKSPACE_TOO_SMALL;
  const size_t R = (size_t)B * H * S, tba = align_up(R * d * 2);
  // what ringx_attn_block_fwd left in its workspace: q | k | v | o | lse
  const char* f = static_cast<const char*>(fwd_workspace);
  const void *q = f, *k = f + tba, *v = f + 2 * tba, *o = f + 3 * tba;
  const float* lse = reinterpret_cast<const float*>(f + 4 * tba);
  char* p = static_cast<char*>(workspace);
  void *d_o = p, *dq = p + tba, *dk = p + 2 * tba, *dv = p + 3 * tba;
  char* inner = p + 4 * tba;
  const size_t inner_bytes = workspace_bytes - 4 * tba;
  st = ringx_out_proj_bwd(dy, o, w_o, d_o, dw_o, B, S, H, d, stream_);
  if (st != RINGX_OK) return st;
  int launches = tl_last_launches;
  st = ringx_attn_bwd(q, k, v, o, lse, d_o, dq, dk, dv, B, H, S, d, kv_chunk, scale, RINGX_BF16, inner, inner_bytes, stream_);
  if (st != RINGX_OK) return st;
  launches += tl_last_launches;
  st = ringx_qkv_proj_bwd(dq, dk, dv, x, w_qkv, dx, dw_qkv, B, S, H, d, stream_);
  if (st != RINGX_OK) return st;
  tl_last_launches += launches;
  return RINGX_OK;
}

// ---- the Turbulence-Transformer tokeniser
int ringx_fidelity_tokens(const float* y, void* tokens, int M, int D, int H, int W, int C, int z0, int y0, int x0,
                          int Dc, int Hc, int Wc, int k, float sigma, int out_dtype, void* stream_) {
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  if (out_dtype != RINGX_F32 && out_dtype != RINGX_BF16) return RINGX_ERR_BAD_DTYPE;
  if (C != 4 || M <= 0 || D <= 0 || H <= 0 || W <= 0 || k < 1 || k > 32) return RINGX_ERR_BAD_SHAPE;
  if (Dc <= 0 || Hc <= 0 || Wc <= 0 || Dc % k || Hc % k || Wc % k) return RINGX_ERR_BAD_SHAPE;
  if (z0 < 0 || y0 < 0 || x0 < 0 || (long long)z0 + Dc > D || (long long)y0 + Hc > H || (long long)x0 + Wc > W)
    return RINGX_ERR_BAD_SHAPE;
  if (Hc / k > 65535 * 1 || (long long)M * (Dc / k) > 65535) return RINGX_ERR_BAD_SHAPE;
  if (!(sigma == sigma) || sigma > 3.0e38f) return RINGX_ERR_BAD_SHAPE;
  if (!y || !tokens) return RINGX_ERR_NULL_PTR;
  if (!aligned16(y) || !aligned16(tokens)) return RINGX_ERR_MISALIGNED;
  int st = check_arch();
  if (st != RINGX_OK) return st;
  // normalised 1-D Gaussian weights (the kernel applies w[a] w[b] w[e]); sigma <= 0 selects the LES filter width k
  const double sg = sigma > 0.f ? (double)sigma : (double)k / sqrt(12.0);
  double g[32], sum = 0.0;
  for (int a = 0; a < k; ++a) {
    const double r = a - 0.5 * (k - 1);
    g[a] = exp(-r * r / (2.0 * sg * sg));
    sum += g[a];
  }
  float w[32];
  for (int a = 0; a < k; ++a) w[a] = (float)(g[a] / sum);
  tl_launches = 0;
  cudaError_t e;
  {
    Timed timed(RINGX_PROFILE_TOKENISER, stream);
    e = launch_fidelity_tokens(y, tokens, M, D, H, W, z0, y0, x0, Dc, Hc, Wc, k, w, out_dtype, stream);
  }
  count_launch();
  if (e != cudaSuccess) return cuda_status(e);
  tl_last_launches = tl_launches;
  return RINGX_OK;
}

// ---- Table II's projection GEMMs and the attention block
static int check_proj(int B, int S, int H, int d) {
  if (B <= 0 || S <= 0 || H <= 0) return RINGX_ERR_BAD_SHAPE;
  if (d != 64 && d != 128) return RINGX_ERR_BAD_SHAPE;
  if (S % 128) return RINGX_ERR_BAD_SHAPE;
  if ((long long)B * S > 0x7fffffffll / 2 || (long long)B * S * H > 0x7fffffffll) return RINGX_ERR_BAD_SHAPE;
  return RINGX_OK;
}

int ringx_qkv_proj(const void* x, const void* w_qkv, void* q, void* k, void* v, int B, int S, int H, int d,
                   void* stream_) {
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  int st = check_proj(B, S, H, d);
  if (st != RINGX_OK) return st;
  if (!x || !w_qkv || !q || !k || !v) return RINGX_ERR_NULL_PTR;
  if (!aligned16(x) || !aligned16(w_qkv) || !aligned16(q) || !aligned16(k) || !aligned16(v)) return RINGX_ERR_MISALIGNED;
  if ((st = check_arch()) != RINGX_OK) return st;
  tl_launches = 0;
  cudaError_t e;
  {
    Timed timed(RINGX_PROFILE_PROJ, stream);
    e = launch_qkv_proj(x, w_qkv, q, k, v, B, S, H, d, stream);
  }
  if (e != cudaSuccess) return cuda_status(e);
  tl_last_launches = tl_launches;
  return RINGX_OK;
}

int ringx_out_proj(const void* o, const void* w_o, void* y, int B, int S, int H, int d, void* stream_) {
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  int st = check_proj(B, S, H, d);
  if (st != RINGX_OK) return st;
  if (!o || !w_o || !y) return RINGX_ERR_NULL_PTR;
  if (!aligned16(o) || !aligned16(w_o) || !aligned16(y)) return RINGX_ERR_MISALIGNED;
  if ((st = check_arch()) != RINGX_OK) return st;
  tl_launches = 0;
  cudaError_t e;
  {
    Timed timed(RINGX_PROFILE_PROJ, stream);
    e = launch_out_proj(o, w_o, y, B, S, H, d, stream);
  }
  if (e != cudaSuccess) return cuda_status(e);
  tl_last_launches = tl_launches;
  return RINGX_OK;
}

size_t ringx_attn_block_fwd_workspace_bytes(int B, int S, int H, int d, int kv_chunk) {
  if (check_proj(B, S, H, d) != RINGX_OK) return 0;
  const size_t R = (size_t)B * H * S;
  return 4 * align_up(R * d * 2) + align_up(R * sizeof(float)) +
         align_up(ringx_attn_fwd_workspace_bytes(B, H, S, d, kv_chunk, RINGX_BF16));
}

int ringx_attn_block_fwd(const void* x, const void* w_qkv, const void* w_o, void* y, int B, int S, int H, int d,
                         int kv_chunk, float scale, void* workspace, size_t workspace_bytes, void* stream_) {
  int st = check_proj(B, S, H, d);
  if (st == RINGX_OK) st = check_shape(B, H, S, d, kv_chunk, scale, RINGX_BF16, false);
  if (st != RINGX_OK) return st;
  if (!x || !w_qkv || !w_o || !y || !workspace) return RINGX_ERR_NULL_PTR;
  if (reinterpret_cast<uintptr_t>(workspace) % kAlign) return RINGX_ERR_MISALIGNED;
  if (workspace_bytes < ringx_attn_block_fwd_workspace_bytes(B, S, H, d, kv_chunk)) return RINGX_ERR_WORKSPACE_TOO_SMALL;
  const size_t R = (size_t)B * H * S, tba = align_up(R * d * 2);
  char* p = static_cast<char*>(workspace);
  void *q = p, *k = p + tba, *v = p + 2 * tba, *o = p + 3 * tba;
  float* lse = reinterpret_cast<float*>(p + 4 * tba);
  char* inner = p + 4 * tba + align_up(R * sizeof(float));
  const size_t inner_bytes = workspace_bytes - (size_t)(inner - p);
  st = ringx_qkv_proj(x, w_qkv, q, k, v, B, S, H, d, stream_);
  if (st != RINGX_OK) return st;
  int launches = tl_last_launches;
  st = ringx_attn_fwd(q, k, v, o, lse, B, H, S, d, kv_chunk, scale, RINGX_BF16, inner, inner_bytes, stream_);
  if (st != RINGX_OK) return st;
  launches += tl_last_launches;
  st = ringx_out_proj(o, w_o, y, B, S, H, d, stream_);
  if (st != RINGX_OK) return st;
  tl_last_launches += launches;
  return RINGX_OK;
}

int ringx_set_deterministic(int on) {
  g_deterministic.store(on != 0 ? 1 : 0, std::memory_order_relaxed);
  return RINGX_OK;
}

int ringx_get_deterministic(void) { return g_deterministic.load(std::memory_order_relaxed); }

int ringx_last_launch_count(void) { return tl_last_launches; }

int ringx_profile_enable(int on) {
  tl_prof.on = on != 0;
  tl_prof.kinds.clear();
  return RINGX_OK;
}

int ringx_profile_read(double* ms, int* launches) {
  if (!ms || !launches) return RINGX_ERR_NULL_PTR;
  for (int i = 0; i < RINGX_PROFILE_KINDS; ++i) { ms[i] = 0.0; launches[i] = 0; }
  Profile& p = tl_prof;
  int st = RINGX_OK;
  for (size_t i = 0; i < p.kinds.size(); ++i) {
    float t = 0.f;
    if (cudaEventSynchronize(p.pool[2 * i + 1]) != cudaSuccess ||
        cudaEventElapsedTime(&t, p.pool[2 * i], p.pool[2 * i + 1]) != cudaSuccess) {
      cudaGetLastError();
      st = RINGX_ERR_CUDA;
      continue;
    }
    ms[p.kinds[i]] += t;
    launches[p.kinds[i]] += 1;
  }
  p.kinds.clear();
  return st;
}

const char* ringx_status_string(int status) {
  switch (status) {
    case RINGX_OK: return "ok";
    case RINGX_ERR_NULL_PTR: return "null pointer";
    case RINGX_ERR_BAD_SHAPE: return "unsupported shape or scale (see include/ringx.h, Domain)";
    case RINGX_ERR_BAD_DTYPE: return "unsupported dtype";
    case RINGX_ERR_MISALIGNED: return "pointer not sufficiently aligned";
    case RINGX_ERR_WORKSPACE_TOO_SMALL: return "workspace too small";
    case RINGX_ERR_UNSUPPORTED_ARCH: return "device is not compute capability 10.x (sm_100a)";
    case RINGX_ERR_CUDA: return "CUDA runtime error";
    default: return "unknown status";
  }
}

int ringx_version(void) { return 150; }

}  // extern "C"
