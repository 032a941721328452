// dwkv_internal.h -- structs shared by the host runtime (dwkv_api.cu) and the kernels. Not part of the ABI.
#pragma once
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>

#include "dwkv_layout.cuh"

namespace dwkv {

// One work unit of the split-T scan: a run of blocks of one (sequence, class) inside one page stripe; the same unit
// exists for every (layer, kv head) (the stripe of (l, h) lies (l*H + h) * kPageLhBytes into the page).
struct __align__(16) Unit {
  int64_t page_off;   // byte offset of the page in the arena
  int32_t blk0;       // first block inside the page's (l,h) stripe
  int32_t nblk;       // number of blocks (>= 1)
  int32_t ntok;       // valid tokens in the unit (last block may be partial)
  int16_t cls;        // class id = 2*tier + flag
  int16_t b;          // index of the sequence in this call's seq_ids
  int32_t epart;      // unused (-1)
  int32_t rk;         // rank of the class
};

struct Scan3Params {            // fused persistent decode kernel (dwkv_scan3*.cuh)
  const uint8_t* arena;
  const Unit* units;           // units of all sequences of the call, grouped by sequence, class-ordered inside
  const int32_t* ustart;       // [n_seqs + 1] unit ranges per sequence
  const int4* wentry;          // [n_slices + 1] slice boundaries (segment, unit, sub-block, first partial slot)
  const int32_t* pstart;       // [n_segs + 1] partial-slot ranges per segment (segment = b * LH + lh)
  const __nv_bfloat16* q;      // [n_seqs][Lq][Hq][d]
  const __nv_bfloat16* BK;     // [M][H][r][d]
  const __nv_bfloat16* gK;     // [L][H][d]
  float* part;                 // [n_slots][G][2 + r + d]: (m, l, a[r], e[d]) per query head
  unsigned long long* stamps;  // optional [2 * n_slices]: globaltimer at the end of every warp slice, segments it touched (NULL = off)
  int32_t n_slices, n_segs;
  int32_t layer0, Lq, LH, w;
  int32_t H, G, r, d;
  float cscale;                // softmax_scale * log2(e)
  float zero;                  // 0.0f (an operand the compiler cannot constant-fold)
  int32_t i8;                  // 8-bit coefficient planes (dwkv_layout.cuh)
  int32_t rot;                 // rotation of the block index per warp in the slice numbering (0, or 53 for single-sequence all-layer calls)
};

struct Combine3Params {
  const int32_t* pstart;       // [n_segs + 1]
  const float* part;
  const __nv_bfloat16* BV;     // [M][H][r][d]
  const __nv_bfloat16* gV;     // [L][H][d]
  float* out;                  // [n_seqs][Lq][Hq][d]
  int32_t layer0, Lq, LH, w;
  int32_t H, G, r, d;
};

// per-token destination for the scatter / gather kernels
struct TokDst {
  int64_t page_off;   // page of the token's class
  int32_t blk;        // block inside the page stripe
  int32_t slot;       // slot inside the block (0..31)
  int32_t cls;        // class id
  int32_t ridx;       // index among the flagged tokens of this call (-1 if unflagged)
  int32_t src;        // append/compress: row of the token in k_new / v_new (the table is sorted flagged-first)
  int32_t pad_;
};

struct CacheGeom {
  int32_t L, w, H, G, r, d, n_tiers;
  int32_t tier_rank[4];
  int32_t i8;         // 8-bit coefficient mode (option "coef_int8"; dwkv_layout.cuh)
};

// records the message dwkv_last_error() returns (thread-local, dwkv_api.cu) and returns `code`
int set_error(int code, const std::string& msg);

// kernel launchers (dwkv_combine3.cu, dwkv_cache_ops.cu, dwkv_dense.cu); each returns the number of kernels launched
int scan3_num_slices(int n_sms);
int launch_scan3(const Scan3Params& p, int n_sms, cudaStream_t s, cudaError_t* err);   // 0 = no instance for this shape; *err = launch status
int launch_combine3(const Combine3Params& p, int n_segs, int split /* 1, 4 or 16 warps per (segment, head) */, cudaStream_t s, cudaError_t* err);
int launch_scatter_raw(const uint8_t* arena, const CacheGeom& g, const TokDst* dst, int n,
                       const __nv_bfloat16* coefK, const __nv_bfloat16* coefV,
                       const float* residK, const float* residV, const uint8_t* codeK, const uint8_t* codeV,
                       const __half* scaleK, const __half* scaleV, cudaStream_t s);
// append/compress work description: the tiles (16 tokens of the sorted table) of one (layer, head) as runs of equal cost
struct CompressRuns {
  int32_t n;            // runs used
  int32_t per_lh;       // sum of count * cost
  int32_t count[16];    // tiles in the run
  int32_t cost[16];     // cost of one tile of the run (compress_tile_cost)
};
// relative cost of one tile: fixed part (row loads, stores), per kept rank chunk, reconstruction + quantiser if a token is flagged
inline int compress_tile_cost(bool flagged, int rank_chunks) { return 4 + 2 * rank_chunks + (flagged ? 12 : 0); }
int launch_compress_mma(const uint8_t* arena, const CacheGeom& g, const TokDst* dst, int n, const CompressRuns& runs /* dst is sorted to match */,
                    const __nv_bfloat16* k_new, const __nv_bfloat16* v_new,
                    const __nv_bfloat16* BK, const __nv_bfloat16* BV, const __nv_bfloat16* gK, const __nv_bfloat16* gV,
                    int n_sms, cudaStream_t s);
// basis construction (dwkv_basis.cu): sketch GEMM + one-sided Jacobi; returns the number of kernels launched (0 = no instance)
size_t basis_scratch_bytes(const CacheGeom& g, int n_sketch, int n_split);
int basis_num_splits(const CacheGeom& g, int n, int n_sms);
int launch_build_basis(const CacheGeom& g, int n, const __nv_bfloat16* k_dense, const __nv_bfloat16* v_dense, const __nv_bfloat16* omega,
                       int n_sketch, int n_split, float* part, const __nv_bfloat16* gK, const __nv_bfloat16* gV, __nv_bfloat16* BK,
                       __nv_bfloat16* BV, bool use_umma /* tcgen05 sketch kernel (d = 128) instead of the mma.sync one */, cudaStream_t s);
struct DumpPtrs {
  __nv_bfloat16 *coefK, *coefV;
  uint8_t *codeK, *codeV;
  __half *scaleK, *scaleV;
  float *deqK, *deqV;
};
int launch_gather(const uint8_t* arena, const CacheGeom& g, const TokDst* dst, int n, const DumpPtrs& o, cudaStream_t s);
int launch_probe_error(const float* ref, const float* cmp, float* e, int n_q, int H, int G, int d, float eps, cudaStream_t s);
// router features: per-token attention mass / spike of one (sequence, layer, query vector); dst = all T tokens in order
size_t token_stats_scratch_bytes(const CacheGeom& g, int64_t T);
int launch_token_stats(const uint8_t* arena, const CacheGeom& g, const TokDst* dst, int T, int layer, const __nv_bfloat16* q,
                       const __nv_bfloat16* BK, const __nv_bfloat16* gK, float cscale, float* scratch, float* mass, float* spike, cudaStream_t s);
int launch_gate_check(const __nv_bfloat16* g, int64_t n, int* bad_flag, cudaStream_t s);

}  // namespace dwkv
