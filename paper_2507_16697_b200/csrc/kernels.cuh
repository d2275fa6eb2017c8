// kernels.cuh -- internal launch interface between the C-ABI layer (api.cu) and the kernels.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <math_constants.h>
#include <stdint.h>

#include "../../include/ringx.h"
#include "ptx.cuh"

namespace ringx {

// ---- merge.cu (HBM-bound helpers)
cudaError_t launch_lse_merge(const void* o_a, const float* lse_a, const void* o_b, const float* lse_b, void* o_out,
                             float* lse_out, long long rows, int d, int in_dtype, int out_dtype, cudaStream_t stream);
// Eq. 5 in its N-operand form: num = loc_out * exp(loc_lse - lse_max), den = exp(loc_lse -
// lse_max) for one operand; o = num/den, lse = lse_max + ln(den) after the sums.  fp32 [rows,d] / [rows].
cudaError_t launch_eq5_scale(const float* loc_out, const float* loc_lse, const float* lse_max, float* num, float* den,
                             long long rows, int d, cudaStream_t stream);
cudaError_t launch_eq5_finalize(const float* num, const float* den, const float* lse_max, void* o_out, float* lse_out,
                                long long rows, int d, int out_dtype, cudaStream_t stream);
// Eq. 5 over the `splits` (<= 8) key splits of one chunk pass: parts [splits][rows,d], lses [splits][rows] fp32, and --
// when o_acc != nullptr -- the running (o_acc, lse_acc) as one more operand.  o_out [rows,d] of out_dtype (may alias
// o_acc when fp32: a thread reads its float4 before writing it), lse_out [rows] (may alias lse_acc only when d == 4...
// it must NOT alias lse_acc: other threads of the row still read it).
cudaError_t launch_split_merge(const float* parts, const float* lses, long long rows, int d, int splits,
                               const float* o_acc, const float* lse_acc, void* o_out, float* lse_out, int out_dtype,
                               cudaStream_t stream);
// D = scale * rowsum(dO*O), lse2 = lse * log2(e); zeroes dq_acc when zero_dq.  rows_per_head > 0: D, lse2 are laid out
// [rows / rows_per_head][rows_per_head rounded up to 128] with lse2 = +inf, D = 0 in the padding (ragged sequences: what
// launch_attn_chunk_bwd_sm100 reads); 0: flat [rows].
cudaError_t launch_bwd_preprocess(const void* o, const void* dO, const float* lse, float* D, float* lse2,
                                  float* dq_acc, long long rows, int d, float scale, bool zero_dq,
                                  cudaStream_t stream, long long rows_per_head = 0);
cudaError_t launch_dq_convert(const float* dq_acc, void* dq, long long n, float scale, cudaStream_t stream);
// Deterministic dQ (int32 fixed-point accumulator, merge.cu).  launch_dq_fixed_scale: kvmax [2*BH] (scratch) and the
// per-row scales qs [BH*rows_per_head] from k (rows d_k wide), v (d_v wide) rows [k_off, k_off+nk) of every head, dO
// (d_v wide) and Ds = launch_bwd_preprocess's D buffer of the same rows (rows_per_head given there too: per-head padded
// layout) (2 launches + a memset).  launch_dq_fixed_finish: dq_bf16 = dq_fix / qs (dq_bf16 != nullptr), else dq_acc += dq_fix / qs
// (1 launch).
cudaError_t launch_dq_fixed_scale(const void* k, const void* v, const void* dO, const float* Ds, float* kvmax, float* qs,
                                  int BH, long long rows_per_head, int nk_stride, int k_off, int nk, int d_k, int d_v,
                                  float scale, cudaStream_t stream);
cudaError_t launch_dq_fixed_finish(const int* dq_fix, const float* qs, void* dq_bf16, float* dq_acc, long long rows, int d,
                                   cudaStream_t stream);

// ---- fidelity.cu (the Turbulence-Transformer tokeniser): crop + k^3 Gaussian filter, stride k.
// y [M,D,H,W,4] fp32 -> tokens [M,Dc/k,Hc/k,Wc/k,4] (f32 or bf16); w = k normalised 1-D weights (host array).
cudaError_t launch_fidelity_tokens(const float* y, void* tokens, int M, int D, int H, int W, int z0, int y0, int x0,
                                   int Dc, int Hc, int Wc, int k, const float* w, int out_dtype, cudaStream_t stream);

// ---- proj_sm100.cu (Table II's projection GEMMs; tcgen05, bf16, fp32 accumulate)
// x [B,S,h], w_qkv [3h,h] = [W_q;W_k;W_v] (y = x W^T) -> q,k,v [B,H,S,d];  o [B,H,S,d], w_o [h,h] -> y [B,S,h].
cudaError_t launch_qkv_proj(const void* x, const void* w_qkv, void* q, void* k, void* v, int B, int S, int H, int d,
                            cudaStream_t stream);
cudaError_t launch_out_proj(const void* o, const void* w_o, void* y, int B, int S, int H, int d, cudaStream_t stream);
// Their backward (two GEMMs each: data gradient in bf16, weight gradient reduce-added in fp32 into a zeroed buffer;
// h % 256 == 0).  dO = split(dY W_o), dW_o = dY^T merge(o);  dX = merge[dq|dk|dv] W_qkv, dW_qkv = merge[dq|dk|dv]^T x.
cudaError_t launch_out_proj_bwd(const void* dy, const void* o, const void* w_o, void* d_o, float* dw_o, int B, int S,
                                int H, int d, cudaStream_t stream);
cudaError_t launch_qkv_proj_bwd(const void* dq, const void* dk, const void* dv, const void* x, const void* w_qkv,
                                void* dx, float* dw_qkv, int B, int S, int H, int d, cudaStream_t stream);

// ---- attn_f32_split_sm100.cu (fp32 accuracy on the bf16 tensor cores by a 3-term operand split; config C1)
// One KV-chunk pass, fp32: q [BH,Nq,d], k/v [BH,nk_stride,d] rows [k_off, k_off+nk) -> o_out fp32, lse_out.
cudaError_t launch_attn_chunk_f32(const float* q, const float* k, const float* v, float* o_out, float* lse_out, int BH,
                                  int Nq, int nk_stride, int k_off, int nk, int d, float scale, cudaStream_t stream);

// ---- attn_fwd_sm100.cu (tcgen05 path)
// One KV-chunk pass, bf16 in / fp32 accumulate.  `epilogue` says what happens to (loc_out, loc_lse):
//   0 written to (o_out, lse_out) as fp32 partials          1 loc_out written as bf16 (single-pass final result)
//   2 folded by the two-operand Eq. 5 into the running fp32 (o_acc, lse_acc); o_out == o_acc, lse_out == lse_acc
//   3 folded with (o_acc, lse_acc) and written to (o_out bf16, lse_out): the last pass
enum { kFwdEpiPartial = 0, kFwdEpiFinal = 1, kFwdEpiFold = 2, kFwdEpiFoldFinal = 3 };
// splits > 1 (kFwdEpiPartial only): split z of the grid takes keys [k_off + z*nk/splits, +nk/splits) and writes its
// partials to o_out + z*BH*Nq*d, lse_out + z*BH*Nq (launch_split_merge combines them).
// Any Nq >= 1; nk % 128 != 0 only for the head's last keys (k_off + nk == nk_stride) and with splits == 1: rows and keys
// past the end of a head are read as zeros through [BH][rows][d] tensor maps, the missing keys are masked (kTail
// instantiation), rows past the end are not written.
cudaError_t launch_attn_chunk_fwd_sm100(const void* q, const void* k, const void* v, void* o_out, float* lse_out,
                                        const float* o_acc, const float* lse_acc, int BH, int Nq, int nk_stride,
                                        int k_off, int nk, int d, float scale, int epilogue, int splits,
                                        cudaStream_t stream);

// ---- attn_fwd_mla_sm100.cu (tcgen05 path, d_qk = 192, d_v = 128: multi-head latent attention in its materialised form)
// One KV-chunk pass: q [BH,Nq,192], k [BH,nk_stride,192], v [BH,nk_stride,128]; epilogues as launch_attn_chunk_fwd_sm100
// (o_out / o_acc are [BH,Nq,128]).
cudaError_t launch_attn_chunk_fwd_mla_sm100(const void* q, const void* k, const void* v, void* o_out, float* lse_out,
                                            const float* o_acc, const float* lse_acc, int BH, int Nq, int nk_stride,
                                            int k_off, int nk, float scale, int epilogue, cudaStream_t stream);

// ---- attn_bwd_mla_sm100.cu (tcgen05 path, d_qk = 192, d_v = 128)
// One KV-chunk pass of the backward: q [BH,N,192], dO [BH,N,128], k,dk [BH,nk_stride,192], v,dv [BH,nk_stride,128];
// writes dk,dv rows [k_off, k_off+nk) of every head (bf16), reduce-adds these keys' contribution to dQ into the
// TRANSPOSED fp32 accumulator dq_acc_t [BH,192,N] (zeroed by the caller before the first pass).  N % 64 == 0.
// lse2, D as for launch_attn_chunk_bwd_sm100 (launch_bwd_preprocess with d = 128).  dkv_dtype: RINGX_BF16 or RINGX_F32.
// dq_qs: nullptr, or [BH * N] per-query scales (launch_dq_fixed_scale): dq_acc_t is then an int32 fixed-point accumulator.
cudaError_t launch_attn_chunk_bwd_mla_sm100(const void* q, const void* k, const void* v, const void* dO,
                                            const float* lse2, const float* D, float* dq_acc_t, void* dk, void* dv,
                                            int BH, int N, int nk_stride, int k_off, int nk, float scale,
                                            const float* dq_qs, int dkv_dtype, cudaStream_t stream);
// dq [BH,N,192] bf16 = transpose(dq_acc_t [BH,192,N] fp32), or of the int32 fixed-point accumulator / dq_qs[query]
cudaError_t launch_dq_transpose_convert_mla(const float* dq_acc_t, void* dq, int BH, int N, const float* dq_qs,
                                            cudaStream_t stream);

// ---- attn_bwd_sm100.cu (tcgen05 path)
// One KV-chunk pass of the backward: q,dO [BH,N,d], k,v,dk,dv [BH,nk_stride,d]; writes dk,dv rows
// [k_off, k_off+nk) of every head (bf16, the sum over the N query rows given), reduce-adds these keys'
// contribution to dQ into dq_acc (fp32 [BH,N,d]).
// lse2 = LSE * log2(e) and D = scale * rowsum(dO*O) come from launch_bwd_preprocess.
// dq_qs: nullptr, or [BH * N] per-row scales (launch_dq_fixed_scale): dq_acc is then an int32 fixed-point
// accumulator and the reduce-adds are integer adds -- bit-reproducible dQ in any arrival order.
// dkv_dtype: RINGX_BF16 (dk, dv bf16) or RINGX_F32 (fp32: one device's share of a cross-device sum).
// Any N >= 1 (lse2, D then in launch_bwd_preprocess's per-head padded layout); nk % 128 != 0 only for the head's last keys.
cudaError_t launch_attn_chunk_bwd_sm100(const void* q, const void* k, const void* v, const void* dO, const float* lse2,
                                        const float* D, float* dq_acc, void* dk, void* dv, int BH, int N,
                                        int nk_stride, int k_off, int nk, int d, float scale, const float* dq_qs,
                                        int dkv_dtype, cudaStream_t stream);

// ---- tensor maps (api.cu): 2-D row-major [rows, cols] view, box = {box_cols, box_rows}
enum TmapSwizzle { kSwizzleNone = 0, kSwizzle128B = 1 };
bool make_tmap_2d(CUtensorMap* out, const void* base, CUtensorMapDataType dt, int elem_bytes, uint64_t rows,
                  uint64_t cols, uint32_t box_rows, uint32_t box_cols, TmapSwizzle swz);
// 2-D view whose rows are pitch_cols (>= cols) elements apart: columns >= cols read as zero and are not written
bool make_tmap_2d_pitched(CUtensorMap* out, const void* base, CUtensorMapDataType dt, int elem_bytes, uint64_t rows,
                          uint64_t cols, uint64_t pitch_cols, uint32_t box_rows, uint32_t box_cols, TmapSwizzle swz);
// 3-D view [heads][rows][cols], box = {box_cols, box_rows, 1}: rows past the end of a head read as zero and are not written
bool make_tmap_3d(CUtensorMap* out, const void* base, CUtensorMapDataType dt, int elem_bytes, uint64_t heads, uint64_t rows,
                  uint64_t cols, uint32_t box_rows, uint32_t box_cols, TmapSwizzle swz);

void count_launch(int n = 1);

// ---- per-device state (api.cu).  The C ABI promises that anything cached is cached per DEVICE, not per process
// (SURVEY.md §8(b)): one process may call on several GPUs.
constexpr int kMaxDevices = 64;
// multiprocessors of the current device, cached per device (148 on B200); 148 when no device can be queried
// (the workspace-size queries also run on boxes without a GPU)
int sm_count();
// cudaFuncAttributeMaxDynamicSharedMemorySize, once per (kernel, device): `done` is the call site's own static array.
// The attribute is idempotent, so the unsynchronised flag is a benign race.
template <typename Kern>
inline cudaError_t set_max_dyn_smem_once(Kern kern, int bytes, unsigned char (&done)[kMaxDevices]) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  const bool cacheable = dev >= 0 && dev < kMaxDevices;
  if (cacheable && done[dev]) return cudaSuccess;
  e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
  if (e != cudaSuccess) return e;
  if (cacheable) done[dev] = 1;
  return cudaSuccess;
}

}  // namespace ringx
