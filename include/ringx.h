/* ringx.h -- C ABI of libringx: the single-GPU hot path of RingX sequence-parallel attention
 * (arXiv 2507.16697, "Pixel-Resolved Long-Context Learning for Turbulence at Exascale"),
 * hand-written for NVIDIA B200 (sm_100a: TMA + tcgen05.mma + TMEM).
 *
 * What the path computes (citations are /root/reference/PAPER.md lines):
 *   - exact, non-causal softmax attention  A^s = sum_i Softmax(Q_s . K_i^T) V_i   (Eq. 1, l.89),
 *     evaluated through the log-sum-exp  LSE_s = log sum_i exp(e_i^s), e_i^s = Q_s . K_i^T
 *     (Eq. 3-4, l.124-126);
 *   - split over key/value chunks S_i whose partial results (loc_out_i, loc_lse_i) are combined by
 *       num = sum_i loc_out_i exp(loc_lse_i - lse_max),  den = sum_i exp(loc_lse_i - lse_max),
 *       A = num/den                                              (Eq. 5, l.130-133; l.137, l.143);
 *     on one GPU the "ring" over devices is a loop over KV-chunk passes (RingX_b with the
 *     all-gather replaced by "K,V already resident", l.145);
 *   - the backward pass: dK,dV complete per KV chunk, dQ "accumulated ... over N steps" (l.143).
 *
 * Conventions that hold for every entry point
 *   Layout     All tensors are contiguous [B,H,N,d], d fastest (the head-split layout
 *              (b*a, S, h/a) of Table II, l.188).  lse is [B,H,N] float.
 *   Pointers   Unless a parameter says HOST, every pointer is a DEVICE pointer, 16-byte aligned.
 *   Ownership  The caller owns every buffer.  The library never allocates or frees device
 *              memory and keeps no pointer after a call returns.  Scratch space is the
 *              caller-provided `workspace`, sized by the *_workspace_bytes queries (the one exception:
 *              ringx_attn_fwd_static, whose scratch is a fixed array inside the library image).
 *   Streams    All work is enqueued on `stream` (a cudaStream_t passed as void*; NULL = legacy
 *              default stream).  Calls return after enqueue; there is no host synchronisation
 *              (the *_host entries are the exception: they synchronise `stream` before returning).  Because nothing
 *              is allocated and nothing synchronises, the device entries can be captured into a CUDA graph
 *              (cudaStreamBeginCapture on `stream`) once their first, uncaptured call has set the kernel attributes.
 *              One-time set-up: the first d = 128 backward on each device checks the alignment of the kernel's shared
 *              memory with a one-warp launch on a short-lived stream of the library's own and waits for that launch
 *              (microseconds; `stream` itself is neither used for it nor synchronised).  If `stream` is being captured
 *              at that moment the call returns RINGX_ERR_CUDA before the attention kernel is enqueued (the capture stays
 *              valid; the call's helper launches may already be in it): make the first backward on a device outside a
 *              capture.
 *   Errors     Return value is a ringx_status (0 = RINGX_OK).  Arguments are validated before the
 *              first launch: an error other than RINGX_ERR_CUDA means nothing was enqueued and no
 *              output was touched.  No abort, no printf, no exceptions cross this boundary.
 *   Domain     d in {64, 128}; kv_chunk % 128 == 0.  ringx_attn_fwd / ringx_attn_bwd and their GQA forms
 *              with RINGX_BF16 take ANY sequence length N >= 1 and any kv_chunk <= N rounded up to 128:
 *              there are ceil(N / kv_chunk) passes, the last one over the keys that are left; tiles
 *              that run past the end of a head read zeros (3-D tensor maps), keys past the end are
 *              masked, rows past the end are never written (the *_host entries and the bf16 per-device
 *              steps ringx_attn_chunk_fwd*, ringx_attn_bwd_partial*, and ringx_attn_fwd_mla /
 *              ringx_attn_bwd_mla likewise).  Every other entry (fp32, the MLA per-device steps, the block
 *              entries) needs N % 128 == 0 (N % 256 == 0 for a
 *              bf16 forward: one CTA owns two 128-row query tiles), 0 < kv_chunk <= N and N % kv_chunk == 0
 *              (every device holds an equal chunk S/N, l.128).  Anything else returns
 *              RINGX_ERR_BAD_SHAPE -- never a silently wrong answer.  A device that is not
 *              compute capability 10.x returns RINGX_ERR_UNSUPPORTED_ARCH.
 *   Semantics  Non-causal, no mask, no dropout, no bias.  `scale` multiplies Q.K^T before the
 *              softmax (Eq. 1/4 print no 1/sqrt(d); it is explicit here); it must be finite and
 *              > 0 (anything else: RINGX_ERR_BAD_SHAPE).  lse is the natural-log
 *              LSE of the *scaled* scores.  bf16 outputs are rounded to nearest even once, at the
 *              end; partial results between chunk passes are fp32.
 *   Threads    Functions are re-entrant.
 */
#ifndef RINGX_H_
#define RINGX_H_

#include <stddef.h>

#if defined(__GNUC__)
#define RINGX_API __attribute__((visibility("default")))
#else
#define RINGX_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  RINGX_OK = 0,
  RINGX_ERR_NULL_PTR = 1,
  RINGX_ERR_BAD_SHAPE = 2,
  RINGX_ERR_BAD_DTYPE = 3,
  RINGX_ERR_MISALIGNED = 4,
  RINGX_ERR_WORKSPACE_TOO_SMALL = 5,
  RINGX_ERR_UNSUPPORTED_ARCH = 6,
  RINGX_ERR_CUDA = 7
} ringx_status;

typedef enum { RINGX_F32 = 0, RINGX_BF16 = 1 } ringx_dtype;

/* Forward (Eq. 1 via Eq. 5).  For c = 0 .. N/kv_chunk-1: one chunk pass computes
 * (loc_out_c, loc_lse_c) of every query row against keys [c*kv_chunk, (c+1)*kv_chunk); partials
 * are folded left to right with the two-operand Eq. 5 in fp32 (bf16: in the chunk kernel's epilogue; f32: by
 * ringx_lse_merge's kernel).
 *   q,k,v  [B,H,N,d] of `dtype` (in).   o [B,H,N,d] of `dtype` (out).   lse [B,H,N] float (out).
 *   dtype  RINGX_BF16: tcgen05 tensor-core path, fp32 accumulation (mixed fp32/bf16, l.286).
 *          RINGX_F32 : fp32 accuracy on the bf16 tensor cores: every fp32 operand is split exactly into three bf16 terms
 *                      and the six leading cross products are accumulated in fp32 (max abs error ~1e-6 on O;
 *                      kind::tf32, 10 mantissa bits, would not meet 1e-5).
 *   workspace  >= ringx_attn_fwd_workspace_bytes(...) bytes, 256-byte aligned; may be NULL when
 *              that query returns 0 (kv_chunk == N with bf16 and a grid large enough that the keys of the
 *              pass are not split, see ringx_attn_chunk_fwd_ex).  Contents are scratch. */
RINGX_API int ringx_attn_fwd(const void* q, const void* k, const void* v, void* o, float* lse,
                   int B, int H, int N, int d, int kv_chunk, float scale, int dtype,
                   void* workspace, size_t workspace_bytes, void* stream);

/* Backward of L = sum dO.O (derivative of Eq. 1; data-flow of l.143).  bf16 only, d = 64 or 128.
 * P is recomputed from the saved *global* lse; each KV-chunk pass writes that chunk's dK,dV once
 * (atomic-free: a CTA owns a 128-key tile) and adds its contribution to dQ in an fp32 accumulator
 * ("accumulated ... over N steps"); the order of the dQ sums is not fixed unless ringx_set_deterministic(1).
 *   q,k,v,o,dO [B,H,N,d] bf16 (in), lse [B,H,N] float (in, as written by ringx_attn_fwd).
 *   dq,dk,dv   [B,H,N,d] bf16 (out); must not alias any input.
 *   workspace  >= ringx_attn_bwd_workspace_bytes(...) bytes, 256-byte aligned. */
RINGX_API int ringx_attn_bwd(const void* q, const void* k, const void* v, const void* o, const float* lse,
                   const void* dO, void* dq, void* dk, void* dv,
                   int B, int H, int N, int d, int kv_chunk, float scale, int dtype,
                   void* workspace, size_t workspace_bytes, void* stream);

/* Grouped-query attention (the paper names MHA / GQA / MLA layers as compatible, l.376): `Hq` query heads share
 * `Hkv` key/value heads, Hq % Hkv == 0, query head h attends kv head h / (Hq/Hkv).
 *   q, o, dO, dq [B,Hq,N,d]; lse [B,Hq,N]; k, v, dk, dv [B,Hkv,N,d].  Everything else as ringx_attn_fwd /
 *   ringx_attn_bwd, whose workspace queries (with H = Hq) size the workspace.  Hq == Hkv is exactly those calls.
 * No extra kernels: the Hq/Hkv heads of a group are adjacent in memory, i.e. (Hq/Hkv)*N query rows against N keys;
 * in the backward the CTA that owns a key tile walks all of them, so dk, dv are still written once, atomic-free. */
RINGX_API int ringx_attn_fwd_gqa(const void* q, const void* k, const void* v, void* o, float* lse,
                       int B, int Hq, int Hkv, int N, int d, int kv_chunk, float scale, int dtype,
                       void* workspace, size_t workspace_bytes, void* stream);
RINGX_API int ringx_attn_bwd_gqa(const void* q, const void* k, const void* v, const void* o, const float* lse,
                       const void* dO, void* dq, void* dk, void* dv,
                       int B, int Hq, int Hkv, int N, int d, int kv_chunk, float scale, int dtype,
                       void* workspace, size_t workspace_bytes, void* stream);

/* Multi-head latent attention shapes (l.376 names MHA / GQA / MLA as the layer designs RingX is compatible with).  In its
 * materialised form an MLA layer attends with a score contraction wider than the values: d_qk = 192 (128 + 64 rotary
 * dimensions) and d_v = 128.  The path is the one of ringx_attn_fwd -- Eq. 1 per KV chunk, partials folded left to right by
 * the two-operand Eq. 5 in the chunk kernel's epilogue -- on a kernel laid out for these widths.
 *   q, k [B,H,N,d_qk] bf16 (in); v [B,H,N,d_v] bf16 (in); o [B,H,N,d_v] bf16 (out); lse [B,H,N] float (out).
 *   Domain: d_qk == 192, d_v == 128, dtype RINGX_BF16, any N >= 1, kv_chunk % 128 == 0 (as ringx_attn_fwd).
 *   workspace  >= ringx_attn_fwd_mla_workspace_bytes(...) bytes (0 when kv_chunk == N), 256-byte aligned. */
RINGX_API int ringx_attn_fwd_mla(const void* q, const void* k, const void* v, void* o, float* lse,
                       int B, int H, int N, int d_qk, int d_v, int kv_chunk, float scale, int dtype,
                       void* workspace, size_t workspace_bytes, void* stream);
RINGX_API size_t ringx_attn_fwd_mla_workspace_bytes(int B, int H, int N, int d_qk, int d_v, int kv_chunk);

/* Backward of the same shapes (the derivative of Eq. 1, P recomputed from the saved LSE; data flow of l.143 as for
 * ringx_attn_bwd): per KV chunk dk, dv of the chunk's keys are complete and written once (atomic-free), dq accumulates in
 * fp32 over the chunk passes (order of the sums not fixed) and is rounded to bf16 once at the end.
 *   q, k, dq, dk [B,H,N,d_qk] bf16; v, o, dO, dv [B,H,N,d_v] bf16; lse [B,H,N] float (from ringx_attn_fwd_mla).
 *   Outputs must not alias inputs.  Domain: d_qk == 192, d_v == 128, RINGX_BF16, any N >= 1, kv_chunk % 128 == 0.
 *   workspace >= ringx_attn_bwd_mla_workspace_bytes(...) bytes, 256-byte aligned (D, LSE*log2e and
 *   the fp32 dq accumulator, which the kernel keeps transposed, [B,H,d_qk,N]; + the fixed-point scales of
 *   ringx_set_deterministic, which applies here as it does to ringx_attn_bwd). */
RINGX_API int ringx_attn_bwd_mla(const void* q, const void* k, const void* v, const void* o, const float* lse,
                       const void* dO, void* dq, void* dk, void* dv,
                       int B, int H, int N, int d_qk, int d_v, int kv_chunk, float scale, int dtype,
                       void* workspace, size_t workspace_bytes, void* stream);
RINGX_API size_t ringx_attn_bwd_mla_workspace_bytes(int B, int H, int N, int d_qk, int d_v, int kv_chunk);

/* The per-device RingX steps (l.137-147) for the same widths -- `Nq` local query rows against the `Nk` keys given:
 * ringx_attn_chunk_fwd_mla is ringx_attn_chunk_fwd_ex (one pass in general form: partials, in-place fold, or last fold to
 * bf16; o_acc / o_out are [B,H,Nq,d_v]; no split-KV, no workspace), Nq % 256 == 0, Nk % 128 == 0;
 * ringx_attn_bwd_partial_mla is ringx_attn_bwd_partial_ex with the fp32 dQ accumulator kept TRANSPOSED, dq_acc_t
 * [B,H,d_qk,Nq] (zeroed by the caller before the first step; reduce-added in arbitrary order), dk [B,H,Nk,d_qk] and dv
 * [B,H,Nk,d_v] of dkv_dtype (bf16, or fp32 shares of a cross-device sum), `prepared` != 0 when the workspace already holds
 * D and LSE*log2e of this (o, lse, dO) from an earlier step; workspace >= ringx_attn_bwd_partial_mla_workspace_bytes(B,H,Nq),
 * Nq % 128 == 0;  ringx_dq_finalize_mla writes dq [B,H,Nq,d_qk] bf16 = transpose(dq_acc_t) after the last step (Nq % 128 == 0
 * like the step that fills dq_acc_t; anything else RINGX_ERR_BAD_SHAPE). */
RINGX_API int ringx_attn_chunk_fwd_mla(const void* q, const void* k, const void* v, const float* o_acc, const float* lse_acc,
                             void* o_out, float* lse_out, int B, int H, int Nq, int Nk, int d_qk, int d_v, float scale,
                             int dtype, int o_out_dtype, void* stream);
RINGX_API int ringx_attn_bwd_partial_mla(const void* q, const void* k, const void* v, const void* o, const float* lse,
                               const void* dO, float* dq_acc_t, void* dk, void* dv,
                               int B, int H, int Nq, int Nk, int d_qk, int d_v, float scale, int dtype, int dkv_dtype,
                               int prepared, void* workspace, size_t workspace_bytes, void* stream);
RINGX_API size_t ringx_attn_bwd_partial_mla_workspace_bytes(int B, int H, int Nq);
RINGX_API int ringx_dq_finalize_mla(const float* dq_acc_t, void* dq, int B, int H, int Nq, int d_qk, void* stream);

/* Two-operand Eq. 5, row by row:  m = max(lse_a,lse_b); w_a = exp(lse_a-m); w_b = exp(lse_b-m);
 * o_out = (w_a o_a + w_b o_b)/(w_a+w_b);  lse_out = m + log(w_a+w_b).
 * An operand with lse = -inf has weight 0; both -inf gives o_out = 0, lse_out = -inf; NaN propagates.
 *   o_a,o_b [rows,d] of o_in_dtype; o_out [rows,d] of o_out_dtype; lse_* [rows] float.
 *   o_out may alias o_a (same dtype) and lse_out may alias lse_a: the merge runs in place.
 *   d % 8 == 0, 8 <= d <= 1024; rows >= 0 (rows == 0 is a no-op). */
RINGX_API int ringx_lse_merge(const void* o_a, const float* lse_a, const void* o_b, const float* lse_b,
                    void* o_out, float* lse_out, long long rows, int d,
                    int o_in_dtype, int o_out_dtype, void* stream);

/* One KV-chunk pass on its own: (loc_out, loc_lse) of `Nq` query rows per head against `Nk` keys
 * (l.135) -- the per-device step of RingX_a/RingX_b with Nq != Nk allowed.
 *   q [B,H,Nq,d], k,v [B,H,Nk,d] of `dtype`; loc_out [B,H,Nq,d] FLOAT; loc_lse [B,H,Nq] float.
 *   bf16: any Nq, Nk >= 1 (ragged tiles are zero-filled, masked and never stored); f32: Nq % 128 == 0, Nk % 128 == 0;
 *   d in {64,128}.  No workspace. */
RINGX_API int ringx_attn_chunk_fwd(const void* q, const void* k, const void* v, float* loc_out, float* loc_lse,
                         int B, int H, int Nq, int Nk, int d, float scale, int dtype, void* stream);

/* ringx_attn_chunk_fwd with the two-operand Eq. 5 folded into the kernel's epilogue: attends `Nq` query rows against
 * the `Nk` keys given and folds (loc_out, loc_lse) into the running partial result (o_acc, lse_acc) of the same rows
 * -- one step of RingX_b's local loop (l.145) without the round trip of loc_out through HBM.
 *   q [B,H,Nq,d], k,v [B,H,Nk,d] bf16; o_acc [B,H,Nq,d] FLOAT, lse_acc [B,H,Nq] float: in/out (as written by
 *   ringx_attn_chunk_fwd, ringx_lse_merge or an earlier fold).
 *   o_final, lse_final: both NULL -> the fold is written back to (o_acc, lse_acc) in place;
 *                       both given -> o_final [B,H,Nq,d] bf16 and lse_final receive the folded result (last step),
 *                       (o_acc, lse_acc) are left untouched.
 *   Any Nq, Nk >= 1, d in {64,128}; dtype must be RINGX_BF16.  No workspace. */
RINGX_API int ringx_attn_chunk_fwd_fold(const void* q, const void* k, const void* v, float* o_acc, float* lse_acc,
                              void* o_final, float* lse_final,
                              int B, int H, int Nq, int Nk, int d, float scale, int dtype, void* stream);

/* One pass in its general form, with split-KV.  When a pass has too few query tiles to fill the 148 SMs (B*H*Nq/256 CTAs --
 * the paper's own regime of 2K-64K query tokens per device against a long gathered key sequence, l.262-264) the library splits
 * the Nk keys over up to 8 groups of CTAs and combines the groups' partial results with Eq. 5 -- the same merge, inside one
 * pass -- into exactly what the unsplit pass returns (up to rounding order).  Whether it splits is the library's choice
 * (ringx_attn_chunk_fwd_ex_workspace_bytes returns 0 when it will not); ringx_attn_fwd / ringx_attn_fwd_gqa do the same inside.
 *   o_acc, lse_acc  NULL: (o_out, lse_out) = (loc_out, loc_lse) of these keys;  else the running fp32 accumulator this pass is
 *                   folded with by the two-operand Eq. 5.
 *   o_out, lse_out  result, o_out of o_out_dtype: RINGX_F32 (may be o_acc, lse_acc themselves: in-place fold) or RINGX_BF16
 *                   (the last pass; must not alias the accumulator).
 *   workspace       >= ringx_attn_chunk_fwd_ex_workspace_bytes(...) bytes, 256-byte aligned; may be NULL when that is 0.
 *   bf16 inputs only; any Nq, Nk >= 1 (split-KV needs Nq % 256 == 0 and Nk % 128 == 0, else the pass is not split),
 *   d in {64,128}. */
RINGX_API int ringx_attn_chunk_fwd_ex(const void* q, const void* k, const void* v, const float* o_acc, const float* lse_acc,
                            void* o_out, float* lse_out, int B, int H, int Nq, int Nk, int d, float scale,
                            int dtype, int o_out_dtype, void* workspace, size_t workspace_bytes, void* stream);
RINGX_API size_t ringx_attn_chunk_fwd_ex_workspace_bytes(int B, int H, int Nq, int Nk, int d, int dtype);

/* Per-device backward step of RingX_a / RingX_b (l.143, l.145): the gradient contributions that `Nq` query
 * rows and `Nk` keys of every head exchange, with P recomputed from the *global* lse of those rows (the
 * LSE over ALL keys of the sequence, not only the Nk given here; reading g8 of DESIGN.md).
 *   q, o, dO [B,H,Nq,d] bf16 (in); lse [B,H,Nq] float (in); k, v [B,H,Nk,d] bf16 (in).
 *   dq_acc [B,H,Nq,d] FLOAT, in/out: += sum over the Nk keys of dS_ij K_j (scale included) -- "the gradient
 *          for Q is accumulated ... over N steps"; the caller zeroes it before the first step and casts it
 *          with ringx_dq_finalize after the last.  Summation order is not fixed unless ringx_set_deterministic(1).
 *   dk, dv [B,H,Nk,d] bf16 (out): the sums over the Nq query rows given (complete when the caller holds
 *          every query of the head, otherwise one device's share to be reduced across devices).
 *   Any Nq, Nk >= 1, d in {64,128}; dtype must be RINGX_BF16.
 *   workspace  >= ringx_attn_bwd_partial_workspace_bytes(B,H,Nq,d) bytes, 256-byte aligned. */
RINGX_API int ringx_attn_bwd_partial(const void* q, const void* k, const void* v, const void* o, const float* lse,
                           const void* dO, float* dq_acc, void* dk, void* dv,
                           int B, int H, int Nq, int Nk, int d, float scale, int dtype,
                           void* workspace, size_t workspace_bytes, void* stream);
RINGX_API size_t ringx_attn_bwd_partial_workspace_bytes(int B, int H, int Nq, int d);

/* ringx_attn_bwd_partial in its general form, as the RingX_a / RingX_b schedules call it once per step (l.143, l.145):
 *   dkv_dtype  RINGX_BF16: dk, dv [B,H,Nk,d] bf16 (as ringx_attn_bwd_partial).
 *              RINGX_F32 : dk, dv [B,H,Nk,d] FLOAT -- the fp32 accumulators written unrounded.  A device's dK,dV of a step are
 *              only its SHARE of a sum over devices (reduce / reduce-scatter, l.143, l.145): reducing fp32 shares and
 *              rounding once keeps the single-device accuracy, where bf16 shares would be rounded W times and then summed
 *              in bf16.
 *   prepared   0: the call first forms D_i = dO_i.O_i and the exp2-domain lse of the Nq rows in the workspace.
 *              1: the workspace still holds them from an earlier call with the same (o, lse, dO, scale, shape) -- every
 *              step of one backward after the first: the preprocess runs once per backward, not once per step.
 * Everything else as ringx_attn_bwd_partial. */
RINGX_API int ringx_attn_bwd_partial_ex(const void* q, const void* k, const void* v, const void* o, const float* lse,
                              const void* dO, float* dq_acc, void* dk, void* dv,
                              int B, int H, int Nq, int Nk, int d, float scale, int dtype, int dkv_dtype, int prepared,
                              void* workspace, size_t workspace_bytes, void* stream);

/* dq = bf16(dq_acc), n elements (n % 4 == 0), round to nearest even: closes the accumulation over steps. */
RINGX_API int ringx_dq_finalize(const float* dq_acc, void* dq, long long n, void* stream);

/* Eq. 5 in its N-operand form, as RingX_a uses it across devices (l.130-133, l.137, l.143):
 *   ringx_eq5_scale     one operand's share: w = exp(loc_lse - lse_max); num = w * loc_out; den = w, where
 *                       lse_max is the element-wise max of loc_lse over all operands (the all-reduce(max));
 *                       an operand with loc_lse = -inf has weight 0 and its loc_out is ignored.
 *   ringx_eq5_finalize  after num and den were summed over the operands (the reduce): o = num / den,
 *                       lse = lse_max + log(den); den = 0 gives o = 0, lse = -inf.
 *   loc_out, num [rows,d] float; loc_lse, lse_max, den, lse_out [rows] float; o_out [rows,d] of o_out_dtype.
 *   num may alias loc_out; o_out may alias num when float; lse_out may alias lse_max.  den must not alias
 *   loc_lse or lse_max, and lse_out must not alias den (other threads of the row still read them).
 *   d % 8 == 0, 8 <= d <= 1024; rows >= 0. */
RINGX_API int ringx_eq5_scale(const float* loc_out, const float* loc_lse, const float* lse_max,
                    float* num, float* den, long long rows, int d, void* stream);
RINGX_API int ringx_eq5_finalize(const float* num, const float* den, const float* lse_max,
                       void* o_out, float* lse_out, long long rows, int d, int o_out_dtype, void* stream);

/* The Turbulence-Transformer tokeniser (l.195-199): one fidelity mode F_k(C(Y)) -- a sub-domain selection C of size
 * Dc x Hc x Wc at origin (z0,y0,x0) followed by a Gaussian filter of kernel size k^3 "via convolution", the result
 * lying in R^{Dc/k x Hc/k x Wc/k x 4}; every filtered voxel is one token (patch size 1, l.179):
 *   T[m,z',y',x',c] = sum_{a,b,e<k} G[a,b,e] * Y[m, z0+k z'+a, y0+k y'+b, x0+k x'+e, c]
 * Readings (the paper is silent; DESIGN.md t1-t6): the convolution has stride k and no padding (forced by the output
 * size); G[a,b,e] = w[a]w[b]w[e], w[a] = g[a]/sum(g), g[a] = exp(-(a-(k-1)/2)^2 / (2 sigma^2)); sigma <= 0 selects
 * the LES Gaussian filter of width k, sigma = k/sqrt(12); the crop lies inside the domain (no periodic wrap);
 * "centered at [x_c,y_c,z_c]" means origin = centre - size/2, computed by the caller.  k = 1 is the pure crop
 * (high-fidelity mode); Dc = D etc. with origin 0 is the low-fidelity mode (no crop).
 *   y       [M,D,H,W,C] float, C fastest (in); C must be 4 (V_x, V_y, V_z, P: l.176).  M = number of input states.
 *   tokens  [M,Dc/k,Hc/k,Wc/k,C] of out_dtype (out), x' fastest: the token sequence of length L = M*Dc*Hc*Wc/k^3.
 *   Domain  1 <= k <= 32; Dc,Hc,Wc multiples of k; Hc/k and M*Dc/k <= 65535; anything else RINGX_ERR_BAD_SHAPE.
 *   fp32 arithmetic (k^3 fused multiply-adds per output); one launch; no workspace. */
RINGX_API int ringx_fidelity_tokens(const float* y, void* tokens, int M, int D, int H, int W, int C,
                          int z0, int y0, int x0, int Dc, int Hc, int Wc, int k, float sigma,
                          int out_dtype, void* stream);

/* Table II's projection GEMMs either side of the attention kernel (l.184-190), bf16 operands, fp32 accumulation on
 * tcgen05, bf16 results (mixed fp32/bf16, l.286):
 *   ringx_qkv_proj  "Input to Q/K/V", (b,S,h) x (h,h) three times: [q|k|v] = x W_qkv^T, written directly in the
 *                   head-split layout (b*a, S, h/a) that the attention entry points read.
 *                   x [B,S,h] (in); w_qkv [3h,h] = [W_q; W_k; W_v], output-feature major (y = x W^T, in);
 *                   q,k,v [B,H,S,d] (out), head a = features [a*d, (a+1)*d).  h = H*d.
 *   ringx_out_proj  "Linear Projection", (bS,h) x (h,h): y = merge_heads(o) W_o^T.
 *                   o [B,H,S,d] (in); w_o [h,h] (in); y [B,S,h] (out).
 *   ringx_attn_block_fwd  the block: ringx_qkv_proj -> ringx_attn_fwd -> ringx_out_proj; q,k,v,o,lse live in the
 *                   workspace (>= ringx_attn_block_fwd_workspace_bytes, 256-byte aligned).
 * No bias, no activation (Table II counts none).  Domain: d in {64,128}; S % 128 == 0 (and the attention domain for
 * the block); anything else RINGX_ERR_BAD_SHAPE.  Outputs must not alias inputs.  One launch per GEMM. */
RINGX_API int ringx_qkv_proj(const void* x, const void* w_qkv, void* q, void* k, void* v,
                   int B, int S, int H, int d, void* stream);
RINGX_API int ringx_out_proj(const void* o, const void* w_o, void* y, int B, int S, int H, int d, void* stream);
RINGX_API int ringx_attn_block_fwd(const void* x, const void* w_qkv, const void* w_o, void* y,
                         int B, int S, int H, int d, int kv_chunk, float scale,
                         void* workspace, size_t workspace_bytes, void* stream);
RINGX_API size_t ringx_attn_block_fwd_workspace_bytes(int B, int S, int H, int d, int kv_chunk);

/* Backward of the projections and of the block (the derivative of the GEMMs above; loss L = sum dY * Y):
 *   ringx_out_proj_bwd   dO = split_heads(dY W_o) (bf16 [B,H,S,d]),  dW_o = dY^T merge_heads(o) (float [h,h]).
 *   ringx_qkv_proj_bwd   dX = merge[dq|dk|dv] W_qkv (bf16 [B,S,h]),  dW_qkv = merge[dq|dk|dv]^T x (float [3h,h]).
 *   ringx_attn_block_bwd ringx_out_proj_bwd -> ringx_attn_bwd -> ringx_qkv_proj_bwd.  fwd_workspace is the workspace of the
 *                        ringx_attn_block_fwd call with the same shape arguments, left untouched since (it holds q, k, v, o, lse).
 * Weight gradients are accumulated in fp32: the buffers are zeroed, then split-K partial sums are reduce-added by TMA (their
 * summation order is not fixed: the last bits may differ from run to run).  Two launches per projection, each a tcgen05
 * GEMM whose transposed operands are read MN-major straight from the row-major tensors (no transpose pass).
 * Domain: as the forward entries, and h = H*d a multiple of 256; else RINGX_ERR_BAD_SHAPE. */
RINGX_API int ringx_out_proj_bwd(const void* dy, const void* o, const void* w_o, void* d_o, float* dw_o,
                       int B, int S, int H, int d, void* stream);
RINGX_API int ringx_qkv_proj_bwd(const void* dq, const void* dk, const void* dv, const void* x, const void* w_qkv,
                       void* dx, float* dw_qkv, int B, int S, int H, int d, void* stream);
RINGX_API int ringx_attn_block_bwd(const void* x, const void* w_qkv, const void* w_o, const void* dy,
                         const void* fwd_workspace, void* dx, float* dw_qkv, float* dw_o,
                         int B, int S, int H, int d, int kv_chunk, float scale,
                         void* workspace, size_t workspace_bytes, void* stream);
RINGX_API size_t ringx_attn_block_bwd_workspace_bytes(int B, int S, int H, int d, int kv_chunk);

/* ringx_attn_fwd with HOST buffers (the end-to-end entry): copies q,k,v host->device into the
 * workspace, runs ringx_attn_fwd, copies o and lse back, and synchronises `stream`.
 *   q_host,k_host,v_host,o_host,lse_host  HOST pointers (pinned memory recommended).
 *   workspace  DEVICE, >= ringx_attn_fwd_host_workspace_bytes(...) bytes. */
RINGX_API int ringx_attn_fwd_host(const void* q_host, const void* k_host, const void* v_host,
                        void* o_host, float* lse_host,
                        int B, int H, int N, int d, int kv_chunk, float scale, int dtype,
                        void* workspace, size_t workspace_bytes, void* stream);

/* Forward + backward with HOST buffers (the end-to-end training-step entry): copies q,k,v,dO host->device
 * into the workspace, runs ringx_attn_fwd then ringx_attn_bwd, copies o, lse, dq, dk, dv back and
 * synchronises `stream`.  bf16 only.  All *_host pointers are HOST pointers (pinned recommended).  The copies overlap the kernels on a
 * side stream the library creates once per thread (a host object; still no device allocation): K,V rows go up chunk by chunk in
 * the order the passes need them, dO goes up during the forward, o and lse come down during the backward, the dK,dV rows of a
 * chunk come down as soon as its pass is done; only dq is copied after the last kernel.
 *   workspace  DEVICE, >= ringx_attn_fwd_bwd_host_workspace_bytes(...) bytes. */
RINGX_API int ringx_attn_fwd_bwd_host(const void* q_host, const void* k_host, const void* v_host,
                            const void* dO_host, void* o_host, float* lse_host,
                            void* dq_host, void* dk_host, void* dv_host,
                            int B, int H, int N, int d, int kv_chunk, float scale, int dtype,
                            void* workspace, size_t workspace_bytes, void* stream);
RINGX_API size_t ringx_attn_fwd_bwd_host_workspace_bytes(int B, int H, int N, int d, int kv_chunk, int dtype);

RINGX_API size_t ringx_attn_fwd_workspace_bytes(int B, int H, int N, int d, int kv_chunk, int dtype);
RINGX_API size_t ringx_attn_bwd_workspace_bytes(int B, int H, int N, int d, int kv_chunk, int dtype);
RINGX_API size_t ringx_attn_fwd_host_workspace_bytes(int B, int H, int N, int d, int kv_chunk, int dtype);

/* ringx_attn_fwd without a workspace argument, for callers that have no device memory to lend and no way to get any.
 * Every other entry point expects the caller to bring the scratch space; some callers cannot:
 *   - a plug-in or operator that runs inside a host process whose own allocator has already claimed the whole GPU
 *     (inference servers and training frameworks reserve HBM up front), where a cudaMalloc simply fails;
 *   - a host thread that must issue work while another thread of the process is capturing a CUDA graph in global capture
 *     mode, during which cudaMalloc is a prohibited call;
 *   - a latency-bound loop (in-situ analysis inside a solver's time step) that cannot take the device-wide synchronisation
 *     cudaMalloc and cudaFree imply;
 *   - a small C or Fortran driver on this ABI that has inputs and outputs but no workspace management of its own.
 * For them the scratch of the multi-pass forward -- the running fp32 (o_acc, lse_acc) that the chunk kernel folds each
 * KV-chunk pass into by the two-operand Eq. 5 (l.130-133), plus the per-split partials when a pass is split over its keys --
 * lives in a fixed array inside the library's device image.  This call, and everything below it, makes no cudaMalloc,
 * cudaFree or other allocating call.
 *   q, k, v, o, lse, shapes, dtype, scale, stream: exactly as ringx_attn_fwd; the results are those of ringx_attn_fwd (same
 *   kernels, same launch configuration, same passes).  Inputs and outputs are still the caller's buffers.
 *   Limit     ringx_attn_fwd_workspace_bytes(B,H,N,d,kv_chunk,dtype) must not exceed RINGX_STATIC_SCRATCH_BYTES (32 MiB:
 *             e.g. B*H*N*d <= 8 Mi elements of fp32 accumulator less the [B,H,N] lse, when no pass is split).  A larger
 *             problem returns RINGX_ERR_WORKSPACE_TOO_SMALL before anything is enqueued -- use ringx_attn_fwd with your
 *             own workspace for those.  A single-pass call (kv_chunk >= N, no split) needs no scratch and always fits.
 *   Cost      the array is part of the library image: every GPU on which the process uses libringx holds those 32 MiB from
 *             module load until the process exits, whether or not this entry is ever called.
 *   Set-up    the first call on each device that needs the scratch looks up the array's device address
 *             (cudaGetSymbolAddress, with that device current; the result is cached per device under a mutex).  Make that
 *             first call outside any stream capture.  A failed look-up returns RINGX_ERR_CUDA.
 *   Sharing   there is ONE array per device and every call uses it.  It keeps whatever the previous call wrote; the forward
 *             needs none of it to start at zero (the first pass overwrites what later passes read), so nothing is cleared.
 *             Two calls whose kernels can overlap on the same GPU -- different streams, or different host threads on different
 *             streams -- race on the array and corrupt each other's results: serialise them (one stream, or an event between
 *             them).  Calls on different GPUs do not interact. */
#define RINGX_STATIC_SCRATCH_BYTES ((size_t)32 << 20)
RINGX_API int ringx_attn_fwd_static(const void* q, const void* k, const void* v, void* o, float* lse,
                          int B, int H, int N, int d, int kv_chunk, float scale, int dtype, void* stream);

/* Bit-reproducible dQ.  By default the per-key-tile contributions to dQ are reduce-added into the fp32
 * accumulator in whatever order the CTAs reach them (fp32 addition is not associative: the last bits of dq may differ from run
 * to run; dk, dv are always bit-reproducible).  With the flag set -- it is process-wide, so that a backward issued from another
 * thread (a framework's autograd worker thread) sees it -- ringx_attn_bwd, ringx_attn_bwd_gqa and ringx_attn_bwd_partial[_ex]
 * accumulate dQ as int32 FIXED POINT: query row i gets the scale
 * 1.5e9 / (1.016 scale (||dO_i|| max_j||V_j|| + |dO_i.O_i|) max_jc|K_jc|), maxima over the keys of the call -- a bound on its
 * |dQ_ic| that follows from sum_j P_ij <= 1 and holds for a per-device step too, where O comes from the keys of all devices
 * and the step's own V may be small or zero (two extra launches read K, V and dO once), every fp32 tile contribution
 * is scaled and rounded to an integer, and the reduce-adds are integer adds -- associative, so the same inputs give
 * bit-identical dq in any arrival order, on any grid, with no ordering between CTAs (about 5 % of the backward throughput at
 * d = 128, 10 % at d = 64).  Resolution: 2^-30.5 of that bound per contribution; for diffuse attention over very long
 * sequences, where |dQ| is far below the bound, this is comparable to the final bf16 rounding (measured at B=1 H=8
 * N=262144 d=128 with iid inputs: rel. Frobenius difference to the fp32 accumulator 1.3e-3), otherwise far below it.
 * ringx_attn_bwd_partial[_ex] keeps the caller's fp32 dq_acc: the step's contribution is accumulated in an int32 scratch
 * inside the workspace and added to dq_acc by one element-wise kernel, so a fixed sequence of steps is reproducible; its
 * workspace query returns the larger size while the flag is set (a call with a workspace sized before the flag was set
 * returns RINGX_ERR_WORKSPACE_TOO_SMALL).  ringx_attn_bwd_mla is covered in the same way (per-query scales on the transposed
 * accumulator).  Non-finite inputs: a NaN or Inf in dO_i, O_i, or in the K, V of the call makes row i of dq NaN (as the fp32
 * accumulator would); a non-finite q or lse is NOT detected in this mode (the integer conversion turns NaN into 0).
 * Not covered: ringx_attn_bwd_partial_mla, and the weight gradients of ringx_*_proj_bwd
 * (split-K partial sums are reduce-added in arbitrary order). */
RINGX_API int ringx_set_deterministic(int on);
RINGX_API int ringx_get_deterministic(void);

/* Number of kernel launches the last successful call on this thread enqueued (bench.py's
 * `gpu_launches` claim is counted here, not guessed). */
RINGX_API int ringx_last_launch_count(void);

/* Optional live per-kernel timing on the calling thread (bench.py's roofline figure).  While enabled,
 * every kernel launch the library makes is bracketed by two CUDA events on the caller's stream (the
 * events are host objects created lazily and reused; no device memory is allocated).
 * ringx_profile_read synchronises on the recorded events, adds the elapsed milliseconds and launch
 * counts per kind into ms[RINGX_PROFILE_KINDS] / launches[RINGX_PROFILE_KINDS] (HOST arrays), and
 * forgets the records.  Kinds: attention forward chunk kernel, Eq. 5 merge kernel, attention
 * backward chunk kernel, backward helpers (D_i preprocess and dQ convert), tokeniser, projection GEMMs. */
enum { RINGX_PROFILE_ATTN_FWD = 0, RINGX_PROFILE_MERGE = 1, RINGX_PROFILE_ATTN_BWD = 2, RINGX_PROFILE_BWD_AUX = 3,
       RINGX_PROFILE_TOKENISER = 4, RINGX_PROFILE_PROJ = 5, RINGX_PROFILE_KINDS = 6 };
RINGX_API int ringx_profile_enable(int on);
RINGX_API int ringx_profile_read(double* ms, int* launches);

RINGX_API const char* ringx_status_string(int status);
RINGX_API int ringx_version(void);

#ifdef __cplusplus
}
#endif
#endif /* RINGX_H_ */
