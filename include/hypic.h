/*
 * hypic.h -- C ABI of libhypic.so: the linear-attention hot path of HYPIC (arxiv/paper_2607_01299, C1)
 * on one NVIDIA B200 (sm_100a).
 *
 * Conventions (row convention of BASELINE.json:north_star; the paper writes the transpose, PAPER.md:80-90,
 * DESIGN.md reading A1).  Per attention head:
 *     state S in R^{dv x dk};  token step  S <- S diag(alpha_t);  S <- S + beta_t (v_t - S k_t) k_t^T,
 *     alpha_t = exp(g_t)   (Eq. 2 with Table 1's dense family)
 *     T_C = prod_{t in C} diag(alpha_t)(I - beta_t k_t k_t^T), first token leftmost
 *     E_C = S after the tokens of C, started from S = 0                  ("S_{C|0}")
 *     compose: S <- S T_i + E_i over a request's ordered segment list     (Eq. 4, 182 Eq. 6)
 *
 * General rules for every entry point:
 *   - Every pointer is a DEVICE pointer unless its comment says HOST.  The caller owns every buffer; the
 *     library allocates nothing, keeps no state between calls and never synchronises the host.  Work is
 *     enqueued on `stream` (a cudaStream_t passed as void*; NULL = the legacy default stream).
 *   - All tensors are dense, row-major, innermost dimension last; pointers must be 16-byte aligned.
 *   - Return value: a hypic_status_t as int.  No exceptions, no abort, nothing printed.  Host-visible
 *     arguments are validated BEFORE any CUDA call (so validation errors are returned on a box with no GPU).
 *     Device-side contents (cu_seqlens, seg_ids, cu_segs) are trusted.  Asynchronous device faults surface
 *     at the caller's next synchronisation, as with any kernel launch.
 *   - There is no CPU fallback: without a usable sm_100 device the compute calls return HYPIC_ERR_CUDA.
 */
#ifndef HYPIC_H_
#define HYPIC_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define HYPIC_VERSION 100 /* 0.1.0 */

typedef enum {
  HYPIC_OK = 0,
  HYPIC_ERR_INVALID_ARG = 1, /* null / negative / inconsistent host-visible argument */
  HYPIC_ERR_UNSUPPORTED = 2, /* shape or dtype outside the built envelope (see each call) */
  HYPIC_ERR_WORKSPACE = 3,   /* workspace NULL or smaller than *_workspace() says */
  HYPIC_ERR_CUDA = 4,        /* a CUDA runtime/driver call failed (no device, launch error, ...) */
  HYPIC_ERR_STATIC_SCRATCH = 5 /* hypic_segment_encode_static: the problem needs more scratch than the built-in array */
} hypic_status_t;

typedef enum { HYPIC_DT_F32 = 0, HYPIC_DT_BF16 = 1 } hypic_dtype_t;          /* dtype of k and v */
typedef enum { HYPIC_GATE_SCALAR = 0, HYPIC_GATE_CHANNEL = 1 } hypic_gate_t; /* g:[Ttot,H] or [Ttot,H,dk] */

/* Kernel families behind the two operations.  AUTO picks the fastest one built for the shape. */
typedef enum {
  HYPIC_IMPL_AUTO = 0,
  HYPIC_IMPL_SIMT = 1,   /* fp32 CUDA-core kernels: token-by-token scan / FFMA compose; any dk in {64,128} */
  HYPIC_IMPL_TENSOR = 2  /* tcgen05/TMEM kernels (dk = dv = 128; encode: bf16 k/v) */
} hypic_impl_t;

/*
 * hypic_set_impl / hypic_get_impl: process-wide selection of the kernel family (default AUTO).  A forced
 * family that does not cover a call's shape makes that call return HYPIC_ERR_UNSUPPORTED.  This is the only
 * global the library keeps; it exists so that tests can check every kernel family against the oracle.
 */
int hypic_set_impl(int impl);
int hypic_get_impl(void);

/*
 * hypic_segment_encode_workspace: bytes of device scratch hypic_segment_encode needs for these arguments
 * (0 is possible).  Returns 0 for arguments the encode call would reject.  Pure host arithmetic.
 */
size_t hypic_segment_encode_workspace(int32_t n_seg, int32_t t_total, int32_t H, int32_t dk, int32_t dv,
                                      int kv_dtype, int gate);

/*
 * hypic_segment_encode: for every segment s (tokens [cu_seqlens[s], cu_seqlens[s+1])) and head h, the
 * zero-start end-state E[s,h] = S_{C|0} (dv x dk) and the segment-cumulative transition
 * T[s,h] = T_C (dk x dk; Eq. 4), both from one pass over the segment's tokens.
 *
 *   k        [t_total, H, dk]   kv_dtype (bf16 or fp32), packed by cu_seqlens
 *   v        [t_total, H, dv]   kv_dtype
 *   g        [t_total, H] (HYPIC_GATE_SCALAR, GDN) or [t_total, H, dk] (HYPIC_GATE_CHANNEL, KDA), fp32
 *            log-decay: alpha = exp(g) (Table 1; reading A2)
 *   beta     [t_total, H] fp32
 *   cu_seqlens  int32 [n_seg+1] on the DEVICE, cu[0] = 0, non-decreasing, cu[n_seg] = t_total (trusted)
 *   E        out [n_seg, H, dv, dk] fp32       T   out [n_seg, H, dk, dk] fp32
 *   workspace / workspace_bytes: device scratch of at least hypic_segment_encode_workspace(...) bytes
 *            (may be NULL when that is 0).  Contents are undefined before and after the call.
 *
 * A zero-length segment yields E = 0, T = I.  n_seg = 0 or t_total = 0 with n_seg > 0 are valid.
 * Built envelope (shapes): dk in {64, 128}; dv in [1, 1024] for the SIMT family (fp32 CUDA cores), dv = dk = 128 with
 * bf16 k/v for the tensor family (tcgen05; scalar or per-channel gate), which HYPIC_IMPL_AUTO takes whenever the shape
 * allows.  Values: any finite inputs.  The tensor family computes with 16-bit operands; what those cannot carry -- a
 * per-channel chunk whose log-decay leaves [-9, 0], values or states beyond fp16's range, a scalar-gate unit of more
 * than 8,192 tokens whose T is still representable (sum g > -72: the 16-bit rounding walk would leave the 3e-3 tolerance
 * of T there) -- is detected on the device per (segment, head) unit, and exactly those units are recomputed by the fp32 family inside the same call, on the
 * same stream, with no host synchronisation and no caller action (the scalar gate never enters the 16-bit algebra, so it
 * has no log-decay limit at all).  hypic_envelope_violation_count remains as a diagnostic counter.
 * H, n_seg, lengths arbitrary.  Inputs are only read; E and T are fully overwritten.
 */
int hypic_segment_encode(const void* k, const void* v, const float* g, const float* beta,
                         const int32_t* cu_seqlens, int32_t n_seg, int32_t t_total, int32_t H, int32_t dk,
                         int32_t dv, int kv_dtype, int gate, float* E, float* T, void* workspace,
                         size_t workspace_bytes, void* stream);

/*
 * hypic_segment_encode_static: hypic_segment_encode (same operation, Eq. 8; same arguments, layouts,
 * envelope, results and error codes) for callers that cannot allocate device memory -- code under CUDA graph capture,
 * tight serving loops, harnesses that forbid cudaMalloc.  The call takes NO workspace and allocates nothing (no
 * cudaMalloc / cudaFree / allocating library routine): its scratch is a file-scope device array inside the library of
 * hypic_static_scratch_bytes() = 4 MiB, held by every GPU that loads the library until the process exits.
 *   - HYPIC_ERR_STATIC_SCRATCH when hypic_segment_encode_workspace(...) for these arguments exceeds
 *     hypic_static_scratch_bytes() (the scalar-gate tensor family needs ~1 KB + 8 n_seg H + 8 (t_total / 64 + n_seg)
 *     bytes: ~33 KB for four folded cfg2 layers; the per-channel gate's prep records, 40 KB per chunk and head, do not
 *     fit beyond ~100 chunk-heads -- use hypic_segment_encode with a caller-owned workspace there).  Nothing is launched.
 *   - The array is shared by every call on the device and keeps the previous call's contents; the call's first kernel
 *     clears what must start at zero.  Calls that OVERLAP on the GPU (different streams without ordering between
 *     them) race on it: issue them on one stream, or order the streams with events.  hypic_segment_encode with
 *     caller-owned workspaces has no such restriction.
 *   - The array's device address is looked up once per device (cudaGetSymbolAddress with that device current) on the
 *     first call there; HYPIC_ERR_CUDA (hypic_last_cuda_error) if that fails.
 */
size_t hypic_static_scratch_bytes(void);
int hypic_segment_encode_static(const void* k, const void* v, const float* g, const float* beta,
                                const int32_t* cu_seqlens, int32_t n_seg, int32_t t_total, int32_t H, int32_t dk,
                                int32_t dv, int kv_dtype, int gate, float* E, float* T, void* stream);

/*
 * hypic_compose: for every request r and head h, fold  S <- S T_i + E_i  (Eq. 6, evaluated as
 * the chain of Eq. 4 steps it abbreviates) over the request's ordered list of pool ids
 * seg_ids[cu_segs[r] .. cu_segs[r+1]) starting from S_in[r,h].  Composition is not commutative: the order
 * is the list order.  An empty list copies S_in (or writes zeros).
 *
 *   S_in     [R, H, dv, dk] fp32, or NULL (= zeros)
 *   E_pool   [P, H, dv, dk] fp32        T_pool  [P, H, dk, dk] fp32  (exactly the E/T layout of encode)
 *   seg_ids  int32 [cu_segs[R]] on the DEVICE, values in [0, P) (trusted)
 *   cu_segs  int32 [R+1] on the DEVICE, cu_segs[0] = 0, non-decreasing (trusted)
 *   total_steps  HOST value of cu_segs[R] (>= 0); used only to size the launch / skip empty work
 *   S_out    out [R, H, dv, dk] fp32; may alias S_in exactly (same pointer), no partial overlap
 *
 * Built envelope: dk in {64, 128}, dv in [1, 1024] (SIMT family); dv = dk = 128 (tensor family, which multiplies
 * two-term fp16 splits and assumes finite pools with |T entries| < 4 -- a transition of a stable recurrence has
 * spectral norm <= 1 -- and |S|, |E| below 1e30; other pools: HYPIC_IMPL_SIMT).
 */
int hypic_compose(const float* S_in, const float* E_pool, const float* T_pool, const int32_t* seg_ids,
                  const int32_t* cu_segs, int32_t R, int32_t P, int32_t total_steps, int32_t H, int32_t dk,
                  int32_t dv, float* S_out, void* stream);

/*
 * hypic_compose_f16: hypic_compose over pools stored in fp16 -- the precision the paper keeps its cached tuples in
 * (32 KB per T at dk = dv = 128: Table 3).  Same fold, same argument meaning and error behaviour as
 * hypic_compose; the differences:
 *   E_pool   [P, H, dv, dk] fp16 (IEEE binary16), T_pool [P, H, dk, dk] fp16; S_in / S_out stay fp32
 *   the stored fp16 values are taken as exact inputs (the result is the fp32-accurate fold of THOSE tuples; what is
 *   lost by storing a tuple in fp16 is lost when it is packed, see hypic_tuple_pack_f16)
 * Built envelope: dv = dk = 128 (tcgen05/TMEM kernel only; there is no SIMT variant), |S| below 1e30.
 */
int hypic_compose_f16(const float* S_in, const void* E_pool, const void* T_pool, const int32_t* seg_ids,
                      const int32_t* cu_segs, int32_t R, int32_t P, int32_t total_steps, int32_t H, int32_t dk, int32_t dv,
                      float* S_out, void* stream);

/*
 * hypic_tuple_pack_f16: dst[i] = fp16(src[i]) (round to nearest even; overflow to +-inf, underflow through fp16
 * subnormals to zero, as IEEE conversion does) for i < count: packs the fp32 E / T tensors of hypic_segment_encode into
 * the fp16 pools of hypic_compose_f16.  src fp32 [count], dst fp16 [count], both 16-byte aligned, no overlap.
 */
int hypic_tuple_pack_f16(const float* src, void* dst, size_t count, void* stream);

/*
 * hypic_seam_window: the seam-window step of PAPER.md:232-234 (section 4.3, Fig. 8).  The first w tokens of an
 * interior segment are left out of the cached tuple and, at reuse time, run through the linear layer on the fly from
 * the running state in front of them, which both advances that state and emits every seam token's output for the layer
 * above.  For every request r and head h:  S = S_in[r,h];  for each token t of [cu_tokens[r], cu_tokens[r+1]) in
 * order: one token step of PAPER.md:84 Eq. 2 (the recurrence hypic_segment_encode accumulates; decay, then erase and
 * write), then the read-out of PAPER.md:86-90 taken AFTER that step:  o[t,h,:] = S_t q_t  (the paper's o_i = q_i^T S_i
 * in the row convention);  S_out[r,h] = S after the last token.  Composing the rest of the segment is hypic_compose
 * on S_out.
 *
 *   q, k     [t_total, H, dk]   kv_dtype (bf16 or fp32)        v   [t_total, H, dv]  kv_dtype
 *   g        [t_total, H] (HYPIC_GATE_SCALAR) or [t_total, H, dk] (HYPIC_GATE_CHANNEL) fp32 log-decay, beta [t_total, H] fp32
 *   cu_tokens  int32 [R+1] on the DEVICE, non-decreasing, 0 <= cu_tokens[0], cu_tokens[R] <= t_total (trusted); windows of
 *            any length are accepted (w = 8 is the paper's default); tokens outside every window are ignored
 *   S_in     [R, H, dv, dk] fp32, or NULL (= zeros)            S_out  out [R, H, dv, dk] fp32, may alias S_in exactly
 *   o        out [t_total, H, dv] fp32; rows of tokens outside every window are left untouched
 *
 * An empty window copies S_in to S_out.  fp32 arithmetic on the CUDA cores (the step moves 8 dk bytes of state per 6 w dk
 * flops, so it is bound by HBM, not by arithmetic); there is no tensor-core variant and hypic_set_impl does not affect
 * it.  Built envelope: dk in {64, 128}, dv in [1, 1024]; R, H <= 65535.
 */
int hypic_seam_window(const void* q, const void* k, const void* v, const float* g, const float* beta,
                      const int32_t* cu_tokens, int32_t R, int32_t t_total, int32_t H, int32_t dk, int32_t dv,
                      int kv_dtype, int gate, const float* S_in, float* S_out, float* o, void* stream);

/*
 * hypic_forward_encode: the segment encode folded into the segment's own forward pass ("accumulating T_C
 * is folded into the first segment prefill"): ONE pass over the tokens of every segment, started from the
 * zero state, emits the per-token layer outputs  o[t,h,:] = S_t q_t together with the tuple
 * (E, T) that hypic_segment_encode returns for the same inputs.  Arguments as hypic_segment_encode plus
 *   q  [t_total, H, dk] kv_dtype        o  out [t_total, H, dv] fp32
 * fp32 arithmetic on the CUDA cores (the token recurrence itself, rows of the stacked state [S ; T] in registers): the
 * accurate form, bound by the fp32 pipe at about a tenth of the tensor family's encode rate; a tcgen05 version of
 * this pass is not built.  Built envelope: dk in {64, 128}, dv in [1, 1024]; n_seg, H <= 65535.  No workspace.
 */
int hypic_forward_encode(const void* q, const void* k, const void* v, const float* g, const float* beta,
                         const int32_t* cu_seqlens, int32_t n_seg, int32_t t_total, int32_t H, int32_t dk, int32_t dv,
                         int kv_dtype, int gate, float* o, float* E, float* T, void* stream);

/*
 * Scalar and diagonal families (Table 1; compressed transitions of PAPER.md:188-200 Table 3).
 * T_i = a_i I (RetNet / Lightning-2 with a constant a_i = gamma, Mamba2 with a data-dependent scalar) or diag(g_i)
 * (GLA); u_i = k_i v_i^T (no beta).  Row convention: S <- S diag(a_t) + v_t k_t^T, a_t = exp(g_t) (A2).
 *
 * hypic_diag_encode: per segment and head, E[s,h] = the end state from S = 0 (dv x dk) and tvec[s,h] = prod_t a_t over
 * the segment's tokens: T_C of Table 3 in its stored form -- ONE scalar for HYPIC_GATE_SCALAR, the dk-vector of the
 * diagonal for HYPIC_GATE_CHANNEL.
 *   k [t_total,H,dk], v [t_total,H,dv] kv_dtype; g [t_total,H] or [t_total,H,dk] fp32 log-decay; cu_seqlens as in
 *   hypic_segment_encode; E out [n_seg,H,dv,dk] fp32; tvec out [n_seg,H] or [n_seg,H,dk] fp32.
 * A zero-length segment yields E = 0, tvec = 1.  Built envelope: dk in {64, 128}, dv in [1, 1024] (the pre-weighting
 * inside the kernels only multiplies by factors in (0, 1] when g <= 0).  No workspace.  Kernel family as selected by
 * hypic_set_impl, see hypic_diag_encode_impl_for.
 *
 * hypic_diag_compose: S <- S diag(tvec_i) + E_i (Eq. 6 with Table 3's "element-wise scaling" apply step;
 * HYPIC_GATE_SCALAR: S <- tvec_i S + E_i) over each request's ordered id list; arguments as hypic_compose with
 * t_pool [P,H] or [P,H,dk] fp32 in place of T_pool.  S_out may alias S_in exactly.  Built envelope: dk % 4 == 0,
 * dk, dv <= 1024.
 */
int hypic_diag_encode(const void* k, const void* v, const float* g, const int32_t* cu_seqlens, int32_t n_seg,
                      int32_t t_total, int32_t H, int32_t dk, int32_t dv, int kv_dtype, int gate, float* E, float* tvec,
                      void* stream);
int hypic_diag_compose(const float* S_in, const float* E_pool, const float* t_pool, const int32_t* seg_ids,
                       const int32_t* cu_segs, int32_t R, int32_t P, int32_t total_steps, int32_t H, int32_t dk,
                       int32_t dv, int gate, float* S_out, void* stream);
/*
 * hypic_rope_compose: state RoPE re-rotation (Eq. 7: S_{C|b} = R(b - a) S_{C|a}) for models of the
 * scalar family that apply RoPE to K inside the linear layer.  T_i = t_i I commutes with every rotation, so a zero-start
 * end-state cached from position 0 is valid at any position after one rotation; at reuse time each S_{C_i|0} of Eq. 6 is
 * replaced by R(p_i) S_{C_i|0}, p_i = the segment's global start position in the spliced sequence:
 *     S <- t_i S + E_i R(p_i)^T      over each request's ordered id list
 * Row convention (keys along the dk columns): every ROW of E_i is rotated like a key.  Pairing (reading R1):
 * column c < dk/2 with column c + dk/2, angle p_i * inv_freq[c]:
 *     E'[:, c] = E[:, c] cos - E[:, c + dk/2] sin,    E'[:, c + dk/2] = E[:, c] sin + E[:, c + dk/2] cos.
 *   S_in, E_pool [P,H,dv,dk] fp32, seg_ids, cu_segs, S_out as in hypic_diag_compose; t_pool [P,H] fp32 (scalar family)
 *   pos       int32 [total_steps]   start position of every list entry (same indexing as seg_ids), >= 0
 *   inv_freq  fp32 [dk/2]           angular frequency of pair c in radians per position (e.g. base^(-2c/dk))
 *   workspace device, >= hypic_rope_compose_workspace(total_steps, dk) bytes, 16-byte aligned; holds the cos/sin table
 *             of this call (angles are formed and reduced in fp64: an fp32 product p * w is off by p * 2^-24 rad)
 * Device-side contents (seg_ids, cu_segs, pos) are trusted.  S_out may alias S_in exactly.  Built envelope: dk in
 * {8, 16, 32, 64, 128}, dv in [1, 1024], H, R <= 65535.  HYPIC_ERR_WORKSPACE when the workspace is missing or too small.
 */
size_t hypic_rope_compose_workspace(int32_t total_steps, int32_t dk);
int hypic_rope_compose(const float* S_in, const float* E_pool, const float* t_pool, const int32_t* seg_ids,
                       const int32_t* cu_segs, const int32_t* pos, const float* inv_freq, int32_t R, int32_t P,
                       int32_t total_steps, int32_t H, int32_t dk, int32_t dv, float* S_out, void* workspace,
                       size_t workspace_bytes, void* stream);
/* hypic_rope_compose_f16: the same over end-states stored in fp16 (hypic_tuple_pack_f16 of hypic_diag_encode's E; the
 * paper's cache precision): E_pool [P,H,dv,dk] fp16, taken as exact inputs and widened to fp32 before
 * the rotation; everything else as hypic_rope_compose. */
int hypic_rope_compose_f16(const float* S_in, const void* E_pool, const float* t_pool, const int32_t* seg_ids,
                           const int32_t* cu_segs, const int32_t* pos, const float* inv_freq, int32_t R, int32_t P,
                           int32_t total_steps, int32_t H, int32_t dk, int32_t dv, float* S_out, void* workspace,
                           size_t workspace_bytes, void* stream);
/* hypic_diag_compose_f16: hypic_diag_compose over end-states stored in fp16 (hypic_tuple_pack_f16 of hypic_diag_encode's
 * E; the paper's cache precision): E_pool [P,H,dv,dk] fp16, taken as exact inputs; t_pool stays fp32
 * (4 B or 4 dk B per tuple: there is nothing to save, and a decay product rounded to fp16 would cost 5e-4 per step). */
int hypic_diag_compose_f16(const float* S_in, const void* E_pool, const float* t_pool, const int32_t* seg_ids,
                           const int32_t* cu_segs, int32_t R, int32_t P, int32_t total_steps, int32_t H, int32_t dk,
                           int32_t dv, int gate, float* S_out, void* stream);
/* hypic_diag_encode_impl_for: as hypic_encode_impl_for, for hypic_diag_encode.  The tcgen05 kernels cover bf16 k/v at
 * dk = dv = 128 for both gates; like the dense tensor family they compute with fp16 operands (finite |k|, |v| <= 65504,
 * g <= 0 so that every weight is <= 1; result within 3e-3 of the oracle, tvec within 1e-5); everything else, and
 * HYPIC_IMPL_SIMT, runs the fp32 CUDA-core kernel (1e-5). */
int hypic_diag_encode_impl_for(int32_t H, int32_t dk, int32_t dv, int kv_dtype, int gate);

/*
 * hypic_encode_impl_for / hypic_compose_impl_for: which kernel family (HYPIC_IMPL_SIMT or HYPIC_IMPL_TENSOR)
 * a call with this shape would run under the current hypic_set_impl setting, or a negative hypic_status_t
 * (-HYPIC_ERR_UNSUPPORTED / -HYPIC_ERR_INVALID_ARG) if the call would be rejected.  Pure host arithmetic;
 * bench.py uses it to name the roofline that bounds the kernel it timed.
 */
int hypic_encode_impl_for(int32_t H, int32_t dk, int32_t dv, int kv_dtype, int gate);
int hypic_compose_impl_for(int32_t H, int32_t dk, int32_t dv);

/*
 * hypic_debug_timeout_count: the tensor-family kernels never spin forever on an mbarrier; a wait that expires
 * (a protocol bug, never expected) bumps a device counter instead of hanging the GPU.  This call synchronises
 * the device and returns the counter since library load (0 = healthy; 0xffffffff = the query itself failed).
 * Test / diagnostics only.
 */
unsigned int hypic_debug_timeout_count(void);

/*
 * hypic_envelope_violation_count: diagnostics.  The per-channel tensor-family encode counts the (chunk, head) pairs whose
 * per-channel log-decay leaves [-9, 0] since library load (their units are recomputed in fp32 inside the same call, see
 * hypic_segment_encode; nothing is left to the caller).  The tcgen05 kernels of hypic_diag_encode add to the same
 * counter for every 64-token chunk that holds a positive or non-finite log-decay (their fp16 weights exp(sum of later
 * log-decays) must not exceed 1; Table 1's gates are <= 1, so such inputs are outside the method's range -- that call
 * has no workspace, so there the caller re-runs with HYPIC_IMPL_SIMT).  Synchronises the device; 0 = never;
 * 0xffffffff = the query itself failed.
 */
unsigned int hypic_envelope_violation_count(void);

/* hypic_status_string: static, NUL-terminated description of a status code (never NULL). */
const char* hypic_status_string(int status);

/* hypic_version: HYPIC_VERSION of the built library. */
int hypic_version(void);

/*
 * hypic_last_launch_count: number of kernel launches the most recent compute call on this thread enqueued
 * (bench.py reports it as gpu_launches).  Pure host bookkeeping.
 */
int hypic_last_launch_count(void);

/*
 * hypic_last_cuda_error: the cudaError_t value behind the most recent HYPIC_ERR_CUDA returned on this thread
 * (0 = none since load).  Pure host bookkeeping; diagnostics only.
 */
int hypic_last_cuda_error(void);

#ifdef __cplusplus
}
#endif
#endif /* HYPIC_H_ */
