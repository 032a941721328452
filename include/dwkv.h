/* dwkv.h -- C ABI of the B200-native DepthWeave-KV decode-attention hot path.
 *
 * The library computes decode-time softmax attention directly over the cross-layer low-rank KV cache of
 * DepthWeave-KV (arxiv/paper_2607_06523) without materialising K-hat / V-hat ("reconstructed KV tensors are not
 * written back to global memory").  Cache content follows PAPER.md:47-56, Eq. (1)
 *     X-hat[l,h,t] = A[l,h,t] . B[m(l),h]  +  g . R[l,h,t]
 * in the reading BASELINE.json `north_star` fixes (readings A1-A21):
 *     K-hat[t,:] = gK[l,h,:] * ( sum_{j<r_t} cK[l,h,t,j] * BK[m(l),h,j,:] ) + f_t * deq(RK[l,h,t])      (same for V)
 *     deq(R)[i]  = code[i] * scale[i/16]       int4 two's-complement codes, fp16 scale per group of 16 channels
 *     m(l) = l / group_size ;  query head hq uses kv head hq / (n_q_heads / n_kv_heads)
 *     o[hq,:] = sum_t softmax_t( q[hq,:] . K-hat[t,:] * softmax_scale ) * V-hat[t,:]
 * Basis, coefficients, gates and q are bf16; accumulation is fp32; outputs are fp32.
 *
 * Conventions
 *   - Every pointer argument is caller-owned.  "dev" = device pointer on cfg.device, "host" = host pointer.
 *     The library copies what it keeps (basis, gates) and owns all cache pages.
 *   - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  Calls enqueue work and return;
 *     host arrays are consumed before the call returns.  dwkv_decode_attention never synchronises the host
 *     unless it has to grow a scratch buffer (first call / larger batch).
 *   - Return value: 0 = DWKV_OK, negative = error (see enum).  No exceptions or aborts cross the ABI.
 *     dwkv_last_error() returns a thread-local message for the last non-zero return.
 *   - One cache per handle; a handle is not thread-safe.  seq_ids within one call must be distinct.
 *   - Limits of this build: d_head in {64, 128}; tier ranks multiples of 8, ascending, last == basis rank <= 64;
 *     n_q_heads / n_kv_heads <= 8.
 */
#ifndef DWKV_H_
#define DWKV_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define DWKV_MAX_TIERS 4

enum {
  DWKV_OK = 0,
  DWKV_E_INVALID = -1,  /* bad config / NULL pointer / tier >= n_tiers / bad layer or sequence id            */
  DWKV_E_STATE = -2,    /* append before basis+gates set; basis or gates changed after tokens exist; bad gate  */
  DWKV_E_CAPACITY = -3, /* sequence slots, tokens per sequence, or arena pages exhausted                       */
  DWKV_E_EMPTY = -4,    /* decode on a sequence with no tokens (softmax over nothing); nothing is launched     */
  DWKV_E_CUDA = -5      /* a CUDA runtime call failed; message in dwkv_last_error()                            */
};

typedef struct dwkv_cache dwkv_cache; /* opaque; owned by the library */

typedef struct {
  int32_t n_layers;                  /* L                                                                      */
  int32_t group_size;                /* w layers per depth window; L % w == 0                    */
  int32_t n_kv_heads;                /* H_kv                                                                   */
  int32_t n_q_heads;                 /* H_q, multiple of H_kv, H_q / H_kv <= 8                                 */
  int32_t d_head;                    /* 64 or 128                                                              */
  int32_t n_tiers;                   /* 1..DWKV_MAX_TIERS rank tiers                                           */
  int32_t tier_rank[DWKV_MAX_TIERS]; /* ascending, multiples of 8; tier_rank[n_tiers-1] == basis rank r        */
  int32_t max_seqs;                  /* sequence slots: valid seq ids are 0..max_seqs-1                        */
  int64_t max_tokens_per_seq;        /* capacity per sequence                                                  */
  float softmax_scale;               /* 0 => 1/sqrt(d_head)  (reading A9)                                      */
  int32_t device;                    /* CUDA device ordinal                                                    */
  void* arena;                       /* optional caller-owned device memory for the cache pages (256-B aligned; cleared by dwkv_create) */
  uint64_t arena_bytes;              /* size of `arena`; if arena == NULL: bytes to cudaMalloc (0 => worst case) */
} dwkv_config;

/* Create a cache. *out receives the handle. Errors: INVALID (config), CUDA (allocation). */
int dwkv_create(const dwkv_config* cfg, dwkv_cache** out);

/* Free everything the library owns (synchronises the device first). dwkv_destroy(NULL) is a no-op. */
void dwkv_destroy(dwkv_cache* c);

/* Shared per-(depth window, head) channel bases B^K, B^V: dev bf16 [L/w, H_kv, r, d], rows assumed
 * orthonormal, used as stored. Copied. Errors: STATE if any sequence already holds tokens (reading A19). */
int dwkv_set_basis(dwkv_cache* c, const void* Bk, const void* Bv, void* stream);

/* Build the bases from the dense K/V of a prefill instead of setting them ("we compute a small randomized low-rank
 * sketch of the cached keys and values after prefill"; reading A24): for every (depth window m, kv head h, Z)
 *     S = sum_{l in window m} Omega_j^T (X_l / gate_l)      (n_sketch x d;  X_l = the n rows k_dense[:, l, h, :], j = l - m*w)
 *     B[m,h] = the r right singular vectors of S with the largest singular values, in descending order, each signed so that its
 *              largest-magnitude entry is positive, rounded to bf16
 * and installs them as dwkv_set_basis would. The gates must be set first (gate-normalised space, reading A13).
 *   k_dense, v_dense  dev bf16 [n, L, H_kv, d]     the prefill vectors (the same layout dwkv_append_compress takes)
 *   omega             dev bf16 [w, n_sketch, n]    the random test matrix the method draws (an INPUT: e.g. N(0,1) values), shared by
 *                                                  all windows, heads and Z; omega[j] multiplies layer j of each window
 *   n                 positive multiple of 8;  n_sketch  multiple of 16, r <= n_sketch <= min(80, d)
 * Enqueues on `stream`, no host sync. Errors: STATE (gates not set, or tokens exist), INVALID (sizes), CUDA. */
int dwkv_build_basis(dwkv_cache* c, int32_t n, const void* k_dense, const void* v_dense, const void* omega, int32_t n_sketch,
                     void* stream);

/* Copy the current bases out: dev bf16 [L/w, H_kv, r, d] each. Errors: STATE (no basis yet). */
int dwkv_export_basis(dwkv_cache* c, void* Bk_out, void* Bv_out, void* stream);

/* Per-layer per-channel gates (reading A8): dev bf16 [L, H_kv, d]. Copied. Synchronises `stream` to validate that
 * every entry is finite and non-zero (STATE otherwise). STATE if any sequence already holds tokens. */
int dwkv_set_gates(dwkv_cache* c, const void* gK, const void* gV, void* stream);

/* Append/compress ("projecting the original cache vector onto the current basis"; readings A13, A14):
 * for every new token, layer, kv head and Z in {K,V}:  c = bf16(B[:r_t] . (x / g));  if flagged, the residual
 * e = x - g * (c . B[:r_t]) is quantised to int4 / group 16 / fp16 scale.  Entries go to the pages of class
 * (tier, flag); slot = number of earlier tokens of the sequence in that class.
 *   seq_ids, n_new : host int32 [n_seqs]      k_new, v_new : dev bf16 [sum(n_new), L, H_kv, d], sequences in call order
 *   tier, flag     : host uint8 [sum(n_new)]  (tier index 0..n_tiers-1, residual flag 0/1)
 * Errors: INVALID, STATE (basis/gates not set), CAPACITY (state is unchanged when INVALID / STATE / CAPACITY is returned), CUDA (a CUDA
 * call failed after the routing was committed: the handle is then poisoned, every later append / decode returns STATE; destroy it). */
int dwkv_append_compress(dwkv_cache* c, int32_t n_seqs, const int32_t* seq_ids, const int32_t* n_new,
                         const void* k_new, const void* v_new, const uint8_t* tier, const uint8_t* flag, void* stream);

/* Fused decode attention: q pre-projection into basis space,
 * split-T online-softmax scan over the tier-segregated pages, split-combine + back-projection through B^V and gV.
 *   layer   : 0..L-1, or -1 = all layers in one call
 *   seq_ids : host int32 [n_seqs], distinct
 *   q       : dev bf16 [n_seqs, H_q, d]  (layer >= 0)   or [n_seqs, L, H_q, d]  (layer == -1)
 *   out     : dev fp32, same shape as q; fully overwritten
 * The query attends to all tokens of the sequence present at call time, no mask (reading A10).
 * Errors: INVALID, STATE, EMPTY (some sequence has no tokens; nothing launched), CUDA. */
int dwkv_decode_attention(dwkv_cache* c, int32_t layer, int32_t n_seqs, const int32_t* seq_ids, const void* q,
                          float* out, void* stream);

/* ---- auxiliaries used by tests and bench (not on the hot path) ------------------------------------------------ */

/* Pre-compressed, token-ordered entries of ONE sequence (device pointers). Residual arrays hold rows for the FLAGGED
 * tokens only, in token order. Exactly one residual mode is used when any token is flagged:
 *   mode A: residK/residV fp32 [n_flagged, L, H_kv, d] -> the library quantises them (reading A14, bit-exact)
 *   mode B: codeK/codeV u8 [n_flagged, L, H_kv, d/2], byte i = channel 2i in the low nibble, 2i+1 in the high nibble,
 *           two's complement;  scaleK/scaleV fp16 [n_flagged, L, H_kv, d/16]                            (reading A7) */
typedef struct {
  const void* coefK;  /* bf16 [n, L, H_kv, r]; entries at j >= r_t are ignored */
  const void* coefV;
  const float* residK;
  const float* residV;
  const uint8_t* codeK;
  const uint8_t* codeV;
  const void* scaleK;
  const void* scaleV;
} dwkv_raw_tokens;

int dwkv_append_raw(dwkv_cache* c, int32_t seq_id, int32_t n, const uint8_t* tier /*host*/, const uint8_t* flag /*host*/,
                    const dwkv_raw_tokens* data, void* stream);

/* Token-ordered dump of tokens [t0, t0+n) of one sequence (device pointers; any may be NULL). Synchronous. */
typedef struct {
  uint8_t* tier;  /* [n] */
  uint8_t* flag;  /* [n] */
  int32_t* slot;  /* [n] slot within the token's class */
  void* coefK;    /* bf16 [n, L, H_kv, r], zero beyond r_t */
  void* coefV;
  uint8_t* codeK; /* u8 [n, L, H_kv, d/2] canonical nibble order; zero rows for unflagged tokens */
  uint8_t* codeV;
  void* scaleK;   /* fp16 [n, L, H_kv, d/16]; zero rows for unflagged tokens */
  void* scaleV;
  float* deqK;    /* fp32 [n, L, H_kv, d] dequantised residual code*scale; zero rows for unflagged tokens */
  float* deqV;
} dwkv_token_dump;

int dwkv_export_tokens(dwkv_cache* c, int32_t seq_id, int64_t t0, int64_t n, const dwkv_token_dump* out, void* stream);

/* Drop all tokens of a sequence and return its pages to the pool (cleared: free pages are always all zero, so appends never
 * clear memory; the whole arena, caller-owned or not, is cleared once by dwkv_create). Synchronises the device. */
int dwkv_reset_seq(dwkv_cache* c, int32_t seq_id);

/* Re-tiering of the stored tokens of one sequence (SURVEY.md section 8f NEXT-4 "re-tiering"; "adaptive threshold chosen
 * to satisfy the current memory budget"; reading A29): every token gets the class (new_tier[t], new_flag[t]), which
 * may only LOWER it: new_tier[t] <= tier[t] and new_flag[t] <= flag[t]. A stored coefficient vector is the leading-r_t part of
 * B (x / gate) (reading A13), so a lower tier is the truncation to its leading r' entries -- bit for bit what an append at that tier
 * would have stored -- and a cleared flag drops the int4 residual; raising a token would need its original vector, which is gone.
 * The tokens keep their order; slots are renumbered per class, the records move to pages of their new classes (device-side gather +
 * scatter of the stored bytes, 8-bit coefficient planes re-blocked exactly) and the old pages return to the pool. Enqueues on
 * `stream`. new_tier, new_flag: HOST uint8 [dwkv_seq_len]. Needs free pages for the whole new layout while the old one is still
 * held (CAPACITY otherwise, nothing changed). Errors: INVALID (NULL, a raised tier / flag), STATE (poisoned handle), CAPACITY, CUDA. */
int dwkv_retier_seq(dwkv_cache* c, int32_t seq_id, const uint8_t* new_tier /*host*/, const uint8_t* new_flag /*host*/, void* stream);

/* Attention-output probe, Eq. (3) (reading A25): for one sequence and
 * layer and n_q probed query positions, the attention output over the compressed cache is compared with the output over a
 * "temporarily materialized higher-fidelity cache" the caller provides for that layer:
 *     e[h] = || Attn(Q, K_ref, V_ref) - Attn(Q, K-hat, V-hat) ||_2 / ( || Attn(Q, K_ref, V_ref) ||_2 + eps )
 * with the norms over the G query heads of kv head h, the n_q positions and all channels. Both attentions use the cache's softmax
 * scale and no mask (every probed query attends to all T = dwkv_seq_len tokens, reading A10).
 *   q            dev bf16 [n_q, H_q, d]
 *   K_ref, V_ref dev bf16 [H_kv, T, d]     (head-major: the layout of the dense comparison kernel)
 *   e_out        dev fp32 [H_kv]
 * Runs dwkv_decode_attention and the dense kernel n_q times each plus one reduction, on `stream`; scratch is owned by the
 * handle. Errors: INVALID, STATE (no basis / gates), EMPTY (T = 0), CUDA. */
int dwkv_probe_error(dwkv_cache* c, int32_t layer, int32_t seq_id, int32_t n_q, const void* q, const void* K_ref, const void* V_ref,
                     float eps, float* e_out, void* stream);

/* Number of cached tokens of a sequence (negative = error code). */
int64_t dwkv_seq_len(const dwkv_cache* c, int32_t seq_id);

/* used = sum over tokens of 4*r_t + f_t*2*(d/2+d/8) bytes times L*H_kv (the compressed footprint, pin P13; with option
 * "coef_int8" the coefficient part is 2*(r_t + ceil(r_t/32)): one code byte per coefficient and one exponent byte per 32-column
 * block of a K / V vector);
 * reserved = bytes of arena pages currently allocated to sequences; dense_equiv = tokens * L * H_kv * 2*d*2. */
int dwkv_footprint(const dwkv_cache* c, uint64_t* used_bytes, uint64_t* reserved_bytes, uint64_t* dense_equiv_bytes);

/* Tuning knobs for experiments (bench / tests); see DESIGN.md section 6. Keys:
 *   "time_scan"       1 = bracket the fused decode kernel and the append/compress kernel with CUDA events
 *                     (dwkv_get_stat "scan_ms" / "compress_ms")
 *   "sketch_umma"     dwkv_build_basis: 1 (default) = TMA + tcgen05 sketch kernel for d = 128, 0 = mma.sync kernel
 *   "max_unit_blocks" planner: blocks (of 32 token slots) per work unit, 0 = by "unit_kb"
 *   "unit_kb"         planner: target size of a work unit per (layer, head), KB (default 64 = one page stripe)
 *   "n_slices"        planner: number of warp slices the step is cut into, 0 (default) = one per warp of the persistent grid,
 *                     fewer (2..7 per SM) when the call is so small that a slice would stream less than ~40 KB
 *   "combine_warps"   combine kernel: warps per (segment, query head): 1 or 4; 0 (default) = by the partials per segment
 *   "interleave"      planner: 1 = interleave the classes of a sequence in the work order, 0 = class after class,
 *                     -1 (default) = interleave when G > 4 or the call lists at most four sequences
 *   "cost_coef_pct", "cost_tok", "cost_resid_pct", "flag_cost_pct"   planner cost model (byte-equivalents per coefficient
 *                     byte in %, per token, per residual byte in %, extra weight of flagged classes in %)
 *   "coef_int8"       1 = store the coefficients "in 8-bit blockwise quantized form" (
 *                     DESIGN.md reading A27): per token, per K / V and per block of 32 rank columns, int8 codes with one power-of-two scale 2^e,
 *                     e the smallest integer with max|c| <= 127 * 2^e (>= -126), code = rint(c / 2^e). code * 2^e is exactly a
 *                     bf16 value, so every call keeps its argument types: dwkv_append_raw quantises the bf16 coefficients it is
 *                     given (lossless if they already lie on the grid), dwkv_append_compress quantises the fp32 projection and
 *                     takes the residual against the dequantised coefficients, dwkv_export_tokens returns code * 2^e as bf16,
 *                     dwkv_decode_attention scans the byte planes (its score contraction runs in fp16 in this mode: the projected
 *                     query q~ = scale * log2(e) * B_K (g_K * q) is split hi + lo in fp16 and clamped to +-65504). A block is 32
 *                     consecutive rank columns of a token's vector (ranks 48 / 64: two blocks, two exponent bytes). Needs an empty
 *                     cache (STATE otherwise). 0 (default) = bf16 coefficients.
 * Any change invalidates the cached plan. Errors: INVALID (unknown key). */
int dwkv_set_option(dwkv_cache* c, const char* key, int64_t value);

/* Measurement aid: with option "time_scan" = 1 every dwkv_decode_attention brackets its fused decode kernel (steps a1 + a2)
 * with CUDA events on `stream`; dwkv_get_stat(c, "scan_ms") waits for the last bracket and returns its duration in
 * milliseconds (negative = none recorded / error); the brackets of the last 64 calls are kept, so a caller can run steps back
 * to back and read them afterwards without a synchronise in between: "scan_ms_mean" / "scan_ms_min" = mean / minimum over the
 * calls timed since "time_scan" was last set (at most the last 64), "scan_samples" = how many those are, "scan_ms@i" = sample i of them (0 = oldest). "compress_ms" is the
 * bracket of the append/compress kernel (step a4) of the last dwkv_append_compress. */
/* Plan of the last dwkv_decode_attention (tests): "plan_slices" = warp slices the work was cut into, "plan_slots" = partial records,
 * "plan_segments" = (sequence, layer, kv head) segments. */
double dwkv_get_stat(dwkv_cache* c, const char* key);

/* Kernels launched by this handle since creation (bench's gpu_launches claim). */
int64_t dwkv_launch_count(const dwkv_cache* c);

const char* dwkv_last_error(void);

/* ---- token-conditional router (Eq. (2); reading A26). Host-only, stateless:
 * "operates only on cache metadata". All pointers are HOST memory.
 *   phi        fp32 [n, 4]  the four online features of a token (attention mass, max spike, boundary indicator, probe error)
 *   u          fp32 [4]     router parameter
 *   z_t = ((u0*phi_t0 + u1*phi_t1) + u2*phi_t2) + u3*phi_t3 in fp32 (no FMA contraction); sigma(z) > tau <=> z > logit(tau), so
 *   thresholds are passed in logit space: tau_logit [n_tiers-1] ascending ("three rank levels"), tau_flag_logit for the
 *   residual flag.  tier_t = #{k : z_t > tau_logit[k]},  flag_t = z_t > tau_flag_logit  -- the arrays dwkv_append_compress takes.
 * Errors: INVALID (NULL, n_tiers outside 1..DWKV_MAX_TIERS, thresholds not ascending / NaN). */
int dwkv_route_tokens(int64_t n, const float* phi, const float* u, int32_t n_tiers, const float* tau_logit, float tau_flag_logit,
                      uint8_t* tier, uint8_t* flag);
/* Thresholds "chosen to satisfy the current memory budget", the budget given as the fraction of tokens per tier
 * (tier_frac [n_tiers], low -> high) and the flagged fraction: tau_logit[k-1] = the largest z_t that is not among the
 * ceil(n * sum_{j>=k} tier_frac[j]) highest ones (the product in double; -inf if every token is, +inf if none); tau_flag_logit the same
 * with flag_frac. With distinct z_t the routed counts are exactly those numbers. */
int dwkv_router_thresholds(int64_t n, const float* phi, const float* u, int32_t n_tiers, const float* tier_frac, float flag_frac,
                           float* tau_logit, float* tau_flag_logit);

/* ---- probe-driven controller (reading A28). Host-only state machine; all
 * pointers are HOST memory. One state (delta_m, quiet_m) per depth window m; thresholds live in logit space (reading A26) and
 * tau_m = base + delta_m. One probe interval = one dwkv_controller_step with the Eq. (3) errors dwkv_probe_error returned:
 *     e_m = max of the errors reported for window m (windows without a probe keep their state)
 *     e_m > tol_m  ->  delta_m = max(delta_m - step_down, delta_min), quiet_m = 0                     "the router lowers tau_m"
 *     else quiet_m += 1, and when quiet_m == patience: delta_m = min(delta_m + step_up, delta_max), quiet_m = 0
 *                                                        "below tolerance for several probe intervals, tau_m is increased"
 * fp32, one rounding per operation (bit-exact against the oracle). Because a token's (tier, flag) is shared by all layers and
 * heads (reading A4), dwkv_controller_thresholds returns base + min_m delta_m: the thresholds dwkv_route_tokens applies to NEW
 * tokens. Stored tokens are never re-tiered (their original vectors no longer exist: promotion is impossible).
 * Errors: INVALID (NULL, sizes, negative steps / tolerances, delta_min > 0 or delta_max < 0, window index out of range, NaN error). */
typedef struct dwkv_controller dwkv_controller; /* opaque; owned by the library */
typedef struct {
  int32_t n_windows;     /* L / w                                                                                   */
  int32_t patience;      /* probe intervals below tolerance before tau_m is raised (>= 1)                           */
  float tol_default;     /* tolerance on e_{l,h} for every window ...                                               */
  const float* tol;      /* ... or host fp32 [n_windows] "window-specific tolerance" (copied); NULL = tol_default    */
  float step_down;       /* logit-space decrement of tau_m on a violation (>= 0)                                    */
  float step_up;         /* logit-space increment after `patience` quiet intervals (>= 0)                           */
  float delta_min;       /* bounds of delta_m: delta_min <= 0 <= delta_max                                          */
  float delta_max;
} dwkv_controller_config;
int dwkv_controller_create(const dwkv_controller_config* cfg, dwkv_controller** out);
void dwkv_controller_destroy(dwkv_controller* ctl);
/* window, e: host [n_probes]: depth window (layer / w) and Eq. (3) error of every probed (layer, kv head) of this interval. */
int dwkv_controller_step(dwkv_controller* ctl, int32_t n_probes, const int32_t* window, const float* e);
/* delta: host fp32 [n_windows], quiet: host int32 [n_windows]; either may be NULL. */
int dwkv_controller_state(const dwkv_controller* ctl, float* delta, int32_t* quiet);
/* tau_logit[k] = base_tau_logit[k] + min_m delta_m (k < n_tiers - 1), *tau_flag_logit = base_flag_logit + min_m delta_m. */
int dwkv_controller_thresholds(const dwkv_controller* ctl, int32_t n_tiers, const float* base_tau_logit, float base_flag_logit,
                               float* tau_logit, float* tau_flag_logit);

/* Router features from the decode path ("accumulated attention mass, maximum attention spike"; reading A28):
 * for one sequence, layer and query vector the softmax probabilities p[hq, t] of all T cached tokens over the compressed cache are
 * formed (the same scores the decode kernel uses; nothing is reconstructed), and
 *     mass[t]  += sum_hq p[hq, t]                 spike[t] = max(spike[t], max_hq p[hq, t])
 * so that calling it on every probe step accumulates phi_0 and phi_1 of Eq. (2) on the device. Token order = append order.
 *   q     dev bf16 [H_q, d]        mass, spike   dev fp32 [T], T = dwkv_seq_len (read-modify-write; zero them before the first probe)
 * Enqueues on `stream`; scratch is owned by the handle, and so is the sequence's device-resident token table (where each token lives
 * and its class id), of which a call uploads only the entries of tokens appended since the last probe.
 * Errors: INVALID, STATE (no basis / gates), EMPTY (T = 0), CUDA. */
int dwkv_probe_token_stats(dwkv_cache* c, int32_t layer, int32_t seq_id, const void* q, float* mass, float* spike, void* stream);

/* ---- dense bf16 comparison kernel (BASELINE.json "from-scratch dense-bf16-cache decode kernel")
 * Plain softmax attention over an uncompressed cache. K, V: dev bf16 [n_seqs, L, H_kv, T, d] (all sequences length T);
 * q: dev bf16 [n_seqs, L, H_q, d]; out: dev fp32 [n_seqs, L, H_q, d]; workspace: dev, >= dwkv_dense_workspace_bytes(). */
uint64_t dwkv_dense_workspace_bytes(int32_t n_seqs, int32_t n_layers, int32_t n_q_heads, int32_t d_head, int64_t T);
int dwkv_dense_decode_attention(const void* K, const void* V, const void* q, float* out, void* workspace,
                                int32_t n_seqs, int32_t n_layers, int32_t n_kv_heads, int32_t n_q_heads, int32_t d_head,
                                int64_t T, float softmax_scale, void* stream);

/* Allocation-free variant of dwkv_dense_decode_attention for callers that cannot call cudaMalloc (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid it): same kernels, same arguments minus `workspace`; the split-T partial records go to
 * a file-scope device array of DWKV_DENSE_STATIC_SCRATCH_BYTES inside the library (every GPU that loads the library holds it until
 * the process exits). The call allocates and frees nothing; the first call on a device resolves the array's device address
 * (cudaGetSymbolAddress, with the caller's current device), so make that first call outside a stream capture.
 *   K, V, q, out: device pointers, layouts as above (caller-owned).
 * A call needs n_seqs * n_layers * n_kv_heads * n_splits * G * (2 + d_head) * 4 bytes, n_splits = min(ceil(1776 / (n_seqs * n_layers
 * * n_kv_heads)), ceil(T / 256)) rounded as dwkv_dense_decode_attention does; e.g. the 8B shape (32 layers, 8 kv heads, G = 4,
 * d = 128) at batch 8 and any T needs 4.3 MB. A call that needs more returns DWKV_E_INVALID and dwkv_last_error() names both sizes.
 * All calls on a device share the array and it keeps the last call's contents. Nothing in it has to be cleared (every record a call
 * reads was written by that call), but two calls that overlap on the GPU (different streams, or graphs replayed concurrently) RACE
 * on it: serialise them, or use dwkv_dense_decode_attention with one workspace per stream.
 * Errors: INVALID (NULL, shapes, scratch too small, device ordinal > 63), CUDA. */
#define DWKV_DENSE_STATIC_SCRATCH_BYTES (16u << 20)
int dwkv_dense_decode_attention_static(const void* K, const void* V, const void* q, float* out, int32_t n_seqs, int32_t n_layers,
                                       int32_t n_kv_heads, int32_t n_q_heads, int32_t d_head, int64_t T, float softmax_scale,
                                       void* stream);

#ifdef __cplusplus
}
#endif
#endif /* DWKV_H_ */
