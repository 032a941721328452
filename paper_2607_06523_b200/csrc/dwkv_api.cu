// dwkv_api.cu -- host runtime and C ABI (include/dwkv.h): cache object, page pool, host-side slot routing,
// work-list planner, launch sequencing. No torch types; plain pointers and sizes only.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

#include "../../include/dwkv.h"
#include "dwkv_internal.h"

using namespace dwkv;

namespace {

thread_local std::string g_err;

int fail(int code, const std::string& msg) {
  g_err = msg;
  return code;
}

}  // namespace

namespace dwkv {
int set_error(int code, const std::string& msg) { return fail(code, msg); }
}  // namespace dwkv

namespace {

#define CU_OK(call)                                                                             \
  do {                                                                                          \
    cudaError_t e__ = (call);                                                                   \
    if (e__ != cudaSuccess)                                                                     \
      return fail(DWKV_E_CUDA, std::string(#call) + ": " + cudaGetErrorString(e__));            \
  } while (0)

// growable device buffer (growth frees the old allocation: implicit device synchronisation, rare)
struct DevBuf {
  void* p = nullptr;
  size_t cap = 0;
  cudaError_t reserve(size_t bytes) {
    if (bytes <= cap) return cudaSuccess;
    if (p) cudaFree(p);
    p = nullptr;
    cap = 0;
    size_t want = std::max(bytes, (size_t)4096);
    want = want + want / 4;
    cudaError_t e = cudaMalloc(&p, want);
    if (e == cudaSuccess) cap = want;
    return e;
  }
  // grow to at least `bytes`, keeping the first `keep` bytes (device-to-device copy on `st`, then the old block is freed:
  // cudaFree waits for the copy)
  cudaError_t grow_keep(size_t bytes, size_t keep, cudaStream_t st) {
    if (bytes <= cap) return cudaSuccess;
    size_t want = std::max(std::max(bytes, 2 * cap), (size_t)4096);
    void* q = nullptr;
    cudaError_t e = cudaMalloc(&q, want);
    if (e != cudaSuccess) return e;
    if (p && keep) e = cudaMemcpyAsync(q, p, keep, cudaMemcpyDeviceToDevice, st);
    if (p) cudaFree(p);
    p = q;
    cap = want;
    return e;
  }
  void release() {
    if (p) cudaFree(p);
    p = nullptr;
    cap = 0;
  }
};

// ring of pinned host staging slots; a slot is reused only after the copy that read it has completed
struct StagingRing {
  static constexpr int kSlots = 4;
  void* host[kSlots] = {nullptr, nullptr, nullptr, nullptr};
  size_t cap[kSlots] = {0, 0, 0, 0};
  cudaEvent_t ev[kSlots] = {nullptr, nullptr, nullptr, nullptr};
  bool pending[kSlots] = {false, false, false, false};
  int next = 0;
  cudaError_t acquire(size_t bytes, void** out, int* slot) {
    const int s = next;
    next = (next + 1) % kSlots;
    cudaError_t e;
    if (!ev[s]) {
      e = cudaEventCreateWithFlags(&ev[s], cudaEventDisableTiming);
      if (e != cudaSuccess) return e;
    }
    if (pending[s]) {
      e = cudaEventSynchronize(ev[s]);
      if (e != cudaSuccess) return e;
      pending[s] = false;
    }
    if (bytes > cap[s]) {
      if (host[s]) cudaFreeHost(host[s]);
      host[s] = nullptr;
      cap[s] = 0;
      size_t want = std::max(bytes + bytes / 4, (size_t)65536);
      e = cudaMallocHost(&host[s], want);
      if (e != cudaSuccess) return e;
      cap[s] = want;
    }
    *out = host[s];
    *slot = s;
    return cudaSuccess;
  }
  cudaError_t mark(int slot, cudaStream_t st) {
    cudaError_t e = cudaEventRecord(ev[slot], st);
    if (e == cudaSuccess) pending[slot] = true;
    return e;
  }
  void release() {
    for (int s = 0; s < kSlots; ++s) {
      if (host[s]) cudaFreeHost(host[s]);
      if (ev[s]) cudaEventDestroy(ev[s]);
      host[s] = nullptr;
      ev[s] = nullptr;
    }
  }
};

struct SeqState {
  std::vector<uint8_t> tier, flag;
  std::vector<int32_t> slot;
  int64_t count[kMaxClasses] = {0, 0, 0, 0, 0, 0, 0, 0};
  std::vector<int32_t> pages[kMaxClasses];
  // device-resident token table: entry t = where token t lives (page, block, slot) and its class id (2 * tier + flag), in append
  // order; the probe kernels walk it. Maintained incrementally: a probe uploads only the entries of the tokens appended since the
  // last one (stored tokens never move, except through dwkv_retier_seq / dwkv_reset_seq, which invalidate it).
  DevBuf tok_dev;
  int64_t tok_dev_n = 0;
};

struct Plan3 {                    // plan of the fused persistent decode kernel (dwkv_scan3*.cuh)
  std::vector<int32_t> seq_ids;
  int n_lsel = 0;
  uint64_t version = ~0ull;
  int n_units = 0, n_slices = 0, n_segs = 0, n_slots = 0;
  size_t off_ustart = 0, off_wentry = 0, off_pstart = 0;
  bool valid = false;
  uint64_t opt_epoch = ~0ull;     // planner options the plan was built with (dwkv_set_option bumps the cache's epoch)
  // structure of the cached plan (units without their token counts, sub-blocks per unit): an append that opens no new sub-block
  // leaves the slices, the partial slots and the unit list as they are -- only Unit::ntok changes
  std::vector<Unit> units;
  std::vector<int32_t> unsub;
};

}  // namespace

struct dwkv_cache {
  dwkv_config cfg;
  CacheGeom geom;
  int n_classes = 0;
  ClassLayout cl[kMaxClasses];
  float softmax_scale = 0.f;
  // page pool
  uint8_t* arena = nullptr;
  bool own_arena = false;
  size_t page_bytes = 0;
  int64_t n_pages = 0;
  std::vector<int32_t> free_pages;
  // model constants
  __nv_bfloat16 *BK = nullptr, *BV = nullptr, *gK = nullptr, *gV = nullptr;
  bool basis_set = false, gates_set = false;
  int* d_flag = nullptr;
  // sequences
  std::vector<SeqState> seqs;
  int64_t total_tokens = 0;
  uint64_t version = 0;
  // scratch
  DevBuf part, plan3_dev, tokdst_dev, basis_scratch, probe_ws, retier_ws;
  uint64_t opt_epoch = 0;            // bumped by every dwkv_set_option: a cached plan is reused only under the options it was built with
  std::vector<uint32_t> seq_stamp;   // duplicate-id check of a call in O(n): stamp per sequence slot
  uint32_t stamp_gen = 0;
  int n_sms = 148;
  StagingRing ring;
  Plan3 plan3;
  // options
  int64_t opt_max_unit_blocks = 0;   // 0 = adaptive
  int64_t opt_cost_coef_pct = 80, opt_cost_tok = -1, opt_cost_resid_pct = -1, opt_cost_seg = 65000;   // planner cost model (-1 = by G)
  int64_t opt_interleave = -1;       // planner: 1 = interleave the classes of a sequence, 0 = class after class, -1 = by shape
  int64_t opt_stamps_ptr = 0;        // device pointer [2 * n_slices] u64 for per-warp end stamps + segment counts (measurement aid), 0 = off
  int64_t opt_unit_kb = 64;          // planner: target bytes of a work unit (per layer-head), KB
  int64_t opt_flag_cost_pct = 85;    // planner weight of flagged-class bytes, percent (100 until the residual-K products shared their A operand)
  int64_t opt_n_slices = 0;          // 0 = one slice per warp of the persistent grid
  int64_t opt_time_scan = 0;
  int64_t opt_combine_warps = 0;     // combine kernel: warps per (segment, head): 1 / 4, 0 = by partials per segment
  int64_t opt_sketch_umma = 1;       // basis sketch: 1 = tcgen05 kernel (d = 128), 0 = mma.sync kernel
  static constexpr int kScanRing = 64;   // "time_scan": the last 64 decode kernels are bracketed, read back without a sync in between
  cudaEvent_t ev_scan0[kScanRing] = {}, ev_scan1[kScanRing] = {}, ev_app0 = nullptr, ev_app1 = nullptr;
  int64_t scan_samples = 0;              // decode kernels timed since "time_scan" was last set
  bool app_timed = false;
  int64_t launches = 0;
  // set when a CUDA call failed AFTER the host had committed the routing of an append (slots, pages, counts): the host index and
  // the pages may then disagree, so every later append / decode / probe call refuses with DWKV_E_STATE until the handle is destroyed
  bool poisoned = false;
};

namespace {

int check_seq(const dwkv_cache* c, int32_t s) { return (s >= 0 && s < c->cfg.max_seqs) ? 0 : -1; }

// armed once an append has committed host state; a return before disarm() (a failed upload, memset or launch) poisons the handle
struct PoisonGuard {
  dwkv_cache* c;
  bool armed = false;
  explicit PoisonGuard(dwkv_cache* cache) : c(cache) {}
  ~PoisonGuard() { if (armed) c->poisoned = true; }
  void arm() { armed = true; }
  void disarm() { armed = false; }
};
const char* kPoisonMsg = "an earlier append failed after its routing was committed: the cache is inconsistent, destroy the handle";

int64_t pages_in_use(const dwkv_cache* c) { return c->n_pages - (int64_t)c->free_pages.size(); }

// Capacity / validity check for n new tokens of one sequence; adds the pages it would need to *need_pages.
// `extra` = tokens of the same sequence already accepted earlier in this call (seq ids are distinct, so 0).
int route_check(const dwkv_cache* c, int32_t seq, int32_t n, const uint8_t* tier, const uint8_t* flag, int64_t* need_pages) {
  const SeqState& S = c->seqs[seq];
  if (n < 0) return fail(DWKV_E_INVALID, "negative token count");
  if ((int64_t)S.tier.size() + n > c->cfg.max_tokens_per_seq) return fail(DWKV_E_CAPACITY, "max_tokens_per_seq exceeded");
  int64_t add[kMaxClasses] = {0, 0, 0, 0, 0, 0, 0, 0};
  for (int i = 0; i < n; ++i) {
    if (tier[i] >= c->cfg.n_tiers || flag[i] > 1) return fail(DWKV_E_INVALID, "tier >= n_tiers or flag > 1");
    add[2 * tier[i] + flag[i]]++;
  }
  for (int k = 0; k < c->n_classes; ++k) {
    const int64_t tpp = c->cl[k].tokens_per_page;
    const int64_t have = (int64_t)S.pages[k].size();
    const int64_t want = (S.count[k] + add[k] + tpp - 1) / tpp;
    *need_pages += std::max<int64_t>(0, want - have);
  }
  return DWKV_OK;
}

// Route n new tokens of one sequence to (class, slot) and pages. Host-side integer routing (reading A15):
// slot = number of earlier tokens of the sequence in the same class. Appends TokDst entries to `out`.
// `ridx_base` numbers the flagged tokens of the whole call. route_check must have passed for the whole call.
void route_commit(dwkv_cache* c, int32_t seq, int32_t n, const uint8_t* tier, const uint8_t* flag, int* ridx_base,
                  std::vector<TokDst>* out, std::vector<int32_t>* new_pages) {
  SeqState& S = c->seqs[seq];
  {   // one growth step for the whole call, geometric (an exact reserve per call would copy the vectors at every decode step)
    const size_t want = S.tier.size() + (size_t)n;
    if (want > S.tier.capacity()) {
      const size_t cap = std::max(want, 2 * S.tier.capacity());
      S.tier.reserve(cap); S.flag.reserve(cap); S.slot.reserve(cap);
    }
  }
  // per class: page index and position inside the page of the next slot, advanced without divisions in the token loop
  int64_t pi[kMaxClasses], in_page[kMaxClasses];
  for (int k = 0; k < c->n_classes; ++k) {
    const int64_t tpp = c->cl[k].tokens_per_page;
    pi[k] = S.count[k] / tpp; in_page[k] = S.count[k] % tpp;
  }
  for (int i = 0; i < n; ++i) {
    const int k = 2 * tier[i] + flag[i];
    const int64_t sl = S.count[k]++;
    if (pi[k] >= (int64_t)S.pages[k].size()) {
      const int32_t pg = c->free_pages.back();
      c->free_pages.pop_back();
      S.pages[k].push_back(pg);
      new_pages->push_back(pg);
    }
    TokDst td;
    td.page_off = (int64_t)S.pages[k][pi[k]] * (int64_t)c->page_bytes;
    td.blk = (int32_t)(in_page[k] / kBlockTok);
    td.slot = (int32_t)(in_page[k] % kBlockTok);
    td.cls = k;
    td.ridx = flag[i] ? (*ridx_base)++ : -1;
    td.src = (int32_t)out->size();
    td.pad_ = 0;
    out->push_back(td);
    if (++in_page[k] == c->cl[k].tokens_per_page) { in_page[k] = 0; pi[k]++; }
    S.tier.push_back(tier[i]);
    S.flag.push_back(flag[i]);
    S.slot.push_back((int32_t)sl);
  }
  c->total_tokens += n;
  c->version++;
}

int upload(dwkv_cache* c, DevBuf& dst, const void* src, size_t bytes, cudaStream_t st) {
  CU_OK(dst.reserve(bytes));
  void* h;
  int slot;
  CU_OK(c->ring.acquire(bytes, &h, &slot));
  memcpy(h, src, bytes);
  CU_OK(cudaMemcpyAsync(dst.p, h, bytes, cudaMemcpyHostToDevice, st));
  CU_OK(c->ring.mark(slot, st));
  return DWKV_OK;
}

int upload_to(dwkv_cache* c, void* dptr, const void* src, size_t bytes, cudaStream_t st) {      // through the pinned staging ring
  void* h;
  int slot;
  CU_OK(c->ring.acquire(bytes, &h, &slot));
  memcpy(h, src, bytes);
  CU_OK(cudaMemcpyAsync(dptr, h, bytes, cudaMemcpyHostToDevice, st));
  CU_OK(c->ring.mark(slot, st));
  return DWKV_OK;
}

// where the stored tokens [t0, t0 + n) of a sequence live: the table the gather / token-statistics kernels walk
void stored_token_table(const dwkv_cache* c, const SeqState& S, int64_t t0, int64_t n, std::vector<TokDst>* out) {
  out->resize((size_t)n);
  for (int64_t i = 0; i < n; ++i) {
    const int k = 2 * S.tier[t0 + i] + S.flag[t0 + i];
    const int64_t sl = S.slot[t0 + i], tpp = c->cl[k].tokens_per_page;
    TokDst td;
    td.page_off = (int64_t)S.pages[k][sl / tpp] * (int64_t)c->page_bytes;
    td.blk = (int32_t)((sl % tpp) / kBlockTok);
    td.slot = (int32_t)((sl % tpp) % kBlockTok);
    td.cls = k;
    td.ridx = -1;
    td.src = (int32_t)i;
    td.pad_ = 0;
    (*out)[(size_t)i] = td;
  }
}

// Invariant: every page in `free_pages` is all zero (the kernels rely on unused slots of a page being zero). The arena is cleared
// once at dwkv_create and a page is cleared again when dwkv_reset_seq returns it to the pool, so the append path never clears
// anything (a prefill-sized call used to spend ~0.3 ms on 1 GB of cudaMemsetAsync, a configs[4] step several 16 MB ones).
int zero_pages(dwkv_cache* c, const std::vector<int32_t>& pages, cudaStream_t st) {
  for (int32_t pg : pages) CU_OK(cudaMemsetAsync(c->arena + (size_t)pg * c->page_bytes, 0, c->page_bytes, st));
  return DWKV_OK;
}

}  // namespace

// =================================================================================================================
// C ABI
// =================================================================================================================
extern "C" {

const char* dwkv_last_error(void) { return g_err.c_str(); }

int dwkv_create(const dwkv_config* cfg, dwkv_cache** out) {
  if (!cfg || !out) return fail(DWKV_E_INVALID, "NULL config or out");
  *out = nullptr;
  const dwkv_config& f = *cfg;
  if (f.n_layers <= 0 || f.group_size <= 0 || f.n_layers % f.group_size) return fail(DWKV_E_INVALID, "n_layers % group_size != 0");
  if (f.n_kv_heads <= 0 || f.n_q_heads <= 0 || f.n_q_heads % f.n_kv_heads) return fail(DWKV_E_INVALID, "n_q_heads % n_kv_heads != 0");
  if (f.n_q_heads / f.n_kv_heads > 8) return fail(DWKV_E_INVALID, "n_q_heads / n_kv_heads > 8 not supported");
  if (f.d_head != 64 && f.d_head != 128) return fail(DWKV_E_INVALID, "d_head must be 64 or 128");
  if (f.n_tiers < 1 || f.n_tiers > DWKV_MAX_TIERS) return fail(DWKV_E_INVALID, "n_tiers out of range");
  for (int k = 0; k < f.n_tiers; ++k) {
    if (f.tier_rank[k] <= 0 || f.tier_rank[k] % 8 || f.tier_rank[k] > 64 || f.tier_rank[k] > f.d_head)
      return fail(DWKV_E_INVALID, "tier ranks must be multiples of 8, <= 64 and <= d_head");
    if (k && f.tier_rank[k] <= f.tier_rank[k - 1]) return fail(DWKV_E_INVALID, "tier ranks must ascend");
    if (f.tier_rank[k] == 40 || f.tier_rank[k] == 56) return fail(DWKV_E_INVALID, "tier ranks 40 and 56 are not instantiated");
  }
  if (f.max_seqs <= 0 || f.max_seqs > 32767 || f.max_tokens_per_seq <= 0) return fail(DWKV_E_INVALID, "bad max_seqs / max_tokens_per_seq");
  if ((int64_t)f.n_layers * f.n_kv_heads > 65535) return fail(DWKV_E_INVALID, "n_layers * n_kv_heads > 65535");
  CU_OK(cudaSetDevice(f.device));

  dwkv_cache* c = new dwkv_cache();
  c->cfg = f;
  if (cudaDeviceGetAttribute(&c->n_sms, cudaDevAttrMultiProcessorCount, f.device) != cudaSuccess || c->n_sms <= 0) c->n_sms = 148;
  c->geom.L = f.n_layers; c->geom.w = f.group_size; c->geom.H = f.n_kv_heads; c->geom.G = f.n_q_heads / f.n_kv_heads;
  c->geom.r = f.tier_rank[f.n_tiers - 1]; c->geom.d = f.d_head; c->geom.n_tiers = f.n_tiers;
  for (int k = 0; k < 4; ++k) c->geom.tier_rank[k] = k < f.n_tiers ? f.tier_rank[k] : 0;
  c->geom.i8 = 0;
  c->n_classes = 2 * f.n_tiers;
  for (int k = 0; k < c->n_classes; ++k) c->cl[k] = make_class_layout(f.tier_rank[k >> 1], k & 1, f.d_head);
  c->softmax_scale = f.softmax_scale > 0.f ? f.softmax_scale : 1.0f / std::sqrt((float)f.d_head);
  c->page_bytes = (size_t)f.n_layers * f.n_kv_heads * kPageLhBytes;
  c->seqs.resize(f.max_seqs);

  uint64_t bytes = f.arena_bytes;
  if (f.arena) {
    if ((reinterpret_cast<uintptr_t>(f.arena) & 255) != 0) { delete c; return fail(DWKV_E_INVALID, "arena not 256-byte aligned"); }
    c->arena = (uint8_t*)f.arena;
  } else {
    if (bytes == 0) {   // worst case: every token in the fattest class, plus one partial page per (seq, class)
      const int64_t tpp = c->cl[c->n_classes - 1].tokens_per_page;
      const int64_t per_seq = (f.max_tokens_per_seq + tpp - 1) / tpp + c->n_classes;
      bytes = (uint64_t)per_seq * f.max_seqs * c->page_bytes;
    }
    void* p = nullptr;
    cudaError_t e = cudaMalloc(&p, bytes);
    if (e != cudaSuccess) { delete c; return fail(DWKV_E_CUDA, std::string("cudaMalloc(arena): ") + cudaGetErrorString(e)); }
    c->arena = (uint8_t*)p;
    c->own_arena = true;
  }
  c->n_pages = (int64_t)(bytes / c->page_bytes);
  if (c->n_pages < 1) { if (c->own_arena) cudaFree(c->arena); delete c; return fail(DWKV_E_INVALID, "arena smaller than one page"); }
  c->free_pages.resize(c->n_pages);
  for (int64_t i = 0; i < c->n_pages; ++i) c->free_pages[i] = (int32_t)(c->n_pages - 1 - i);   // pop -> ascending ids
  {   // free pages are all zero (see zero_pages): clear the arena once, here
    cudaError_t ez = cudaMemset(c->arena, 0, (size_t)c->n_pages * c->page_bytes);
    if (ez == cudaSuccess) ez = cudaDeviceSynchronize();
    if (ez != cudaSuccess) { dwkv_destroy(c); return fail(DWKV_E_CUDA, std::string("cudaMemset(arena): ") + cudaGetErrorString(ez)); }
  }

  const size_t nb = (size_t)(f.n_layers / f.group_size) * f.n_kv_heads * c->geom.r * f.d_head * sizeof(__nv_bfloat16);
  const size_t ng = (size_t)f.n_layers * f.n_kv_heads * f.d_head * sizeof(__nv_bfloat16);
  cudaError_t e = cudaMalloc((void**)&c->BK, nb);
  if (e == cudaSuccess) e = cudaMalloc((void**)&c->BV, nb);
  if (e == cudaSuccess) e = cudaMalloc((void**)&c->gK, ng);
  if (e == cudaSuccess) e = cudaMalloc((void**)&c->gV, ng);
  if (e == cudaSuccess) e = cudaMalloc((void**)&c->d_flag, sizeof(int));
  if (e != cudaSuccess) { dwkv_destroy(c); return fail(DWKV_E_CUDA, std::string("cudaMalloc(constants): ") + cudaGetErrorString(e)); }
  *out = c;
  return DWKV_OK;
}

void dwkv_destroy(dwkv_cache* c) {
  if (!c) return;
  cudaSetDevice(c->cfg.device);
  cudaDeviceSynchronize();
  if (c->own_arena && c->arena) cudaFree(c->arena);
  if (c->BK) cudaFree(c->BK);
  if (c->BV) cudaFree(c->BV);
  if (c->gK) cudaFree(c->gK);
  if (c->gV) cudaFree(c->gV);
  if (c->d_flag) cudaFree(c->d_flag);
  for (SeqState& S : c->seqs) S.tok_dev.release();
  c->part.release(); c->plan3_dev.release(); c->tokdst_dev.release(); c->basis_scratch.release(); c->probe_ws.release(); c->retier_ws.release();
  c->ring.release();
  for (int i = 0; i < dwkv_cache::kScanRing; ++i) {
    if (c->ev_scan0[i]) cudaEventDestroy(c->ev_scan0[i]);
    if (c->ev_scan1[i]) cudaEventDestroy(c->ev_scan1[i]);
  }
  if (c->ev_app0) cudaEventDestroy(c->ev_app0);
  if (c->ev_app1) cudaEventDestroy(c->ev_app1);
  delete c;
}

int dwkv_set_basis(dwkv_cache* c, const void* Bk, const void* Bv, void* stream) {
  if (!c || !Bk || !Bv) return fail(DWKV_E_INVALID, "NULL argument");
  if (c->total_tokens > 0) return fail(DWKV_E_STATE, "basis is frozen once tokens exist (reading A19)");
  const size_t nb = (size_t)(c->geom.L / c->geom.w) * c->geom.H * c->geom.r * c->geom.d * sizeof(__nv_bfloat16);
  cudaStream_t st = (cudaStream_t)stream;
  CU_OK(cudaMemcpyAsync(c->BK, Bk, nb, cudaMemcpyDeviceToDevice, st));
  CU_OK(cudaMemcpyAsync(c->BV, Bv, nb, cudaMemcpyDeviceToDevice, st));
  c->basis_set = true;
  return DWKV_OK;
}

int dwkv_build_basis(dwkv_cache* c, int32_t n, const void* k_dense, const void* v_dense, const void* omega, int32_t n_sketch,
                     void* stream) {
  if (!c || !k_dense || !v_dense || !omega) return fail(DWKV_E_INVALID, "NULL argument");
  if (!c->gates_set) return fail(DWKV_E_STATE, "gates must be set before the basis is built (the sketch is taken in gate-normalised space)");
  if (c->total_tokens > 0) return fail(DWKV_E_STATE, "basis is frozen once tokens exist (reading A19)");
  if (n <= 0 || n % 8) return fail(DWKV_E_INVALID, "n must be a positive multiple of 8");
  if (n_sketch % 16 || n_sketch < c->geom.r || n_sketch > 80 || n_sketch > c->geom.d)
    return fail(DWKV_E_INVALID, "n_sketch must be a multiple of 16 with r <= n_sketch <= min(80, d_head)");
  cudaStream_t st = (cudaStream_t)stream;
  const int ns = basis_num_splits(c->geom, n, c->n_sms);
  CU_OK(c->basis_scratch.reserve(basis_scratch_bytes(c->geom, n_sketch, ns)));
  const int launched = launch_build_basis(c->geom, n, (const __nv_bfloat16*)k_dense, (const __nv_bfloat16*)v_dense,
                                          (const __nv_bfloat16*)omega, n_sketch, ns, (float*)c->basis_scratch.p, c->gK, c->gV, c->BK,
                                          c->BV, c->opt_sketch_umma != 0, st);
  if (!launched) return fail(DWKV_E_INVALID, "no sketch kernel instance for this shape");
  c->launches += launched;
  CU_OK(cudaGetLastError());
  c->basis_set = true;
  return DWKV_OK;
}

int dwkv_export_basis(dwkv_cache* c, void* Bk_out, void* Bv_out, void* stream) {
  if (!c || !Bk_out || !Bv_out) return fail(DWKV_E_INVALID, "NULL argument");
  if (!c->basis_set) return fail(DWKV_E_STATE, "no basis set");
  const size_t nb = (size_t)(c->geom.L / c->geom.w) * c->geom.H * c->geom.r * c->geom.d * sizeof(__nv_bfloat16);
  cudaStream_t st = (cudaStream_t)stream;
  CU_OK(cudaMemcpyAsync(Bk_out, c->BK, nb, cudaMemcpyDeviceToDevice, st));
  CU_OK(cudaMemcpyAsync(Bv_out, c->BV, nb, cudaMemcpyDeviceToDevice, st));
  return DWKV_OK;
}

int dwkv_set_gates(dwkv_cache* c, const void* gK, const void* gV, void* stream) {
  if (!c || !gK || !gV) return fail(DWKV_E_INVALID, "NULL argument");
  if (c->total_tokens > 0) return fail(DWKV_E_STATE, "gates are frozen once tokens exist");
  const int64_t n = (int64_t)c->geom.L * c->geom.H * c->geom.d;
  cudaStream_t st = (cudaStream_t)stream;
  CU_OK(cudaMemsetAsync(c->d_flag, 0, sizeof(int), st));
  c->launches += launch_gate_check((const __nv_bfloat16*)gK, n, c->d_flag, st);
  c->launches += launch_gate_check((const __nv_bfloat16*)gV, n, c->d_flag, st);
  int bad = 0;
  CU_OK(cudaMemcpyAsync(&bad, c->d_flag, sizeof(int), cudaMemcpyDeviceToHost, st));
  CU_OK(cudaStreamSynchronize(st));
  if (bad) return fail(DWKV_E_STATE, "gate entries must be finite and non-zero (reading A13)");
  CU_OK(cudaMemcpyAsync(c->gK, gK, n * sizeof(__nv_bfloat16), cudaMemcpyDeviceToDevice, st));
  CU_OK(cudaMemcpyAsync(c->gV, gV, n * sizeof(__nv_bfloat16), cudaMemcpyDeviceToDevice, st));
  c->gates_set = true;
  return DWKV_OK;
}

int dwkv_append_compress(dwkv_cache* c, int32_t n_seqs, const int32_t* seq_ids, const int32_t* n_new, const void* k_new,
                         const void* v_new, const uint8_t* tier, const uint8_t* flag, void* stream) {
  if (!c || n_seqs < 0 || (n_seqs > 0 && (!seq_ids || !n_new))) return fail(DWKV_E_INVALID, "NULL argument");
  if (!c->basis_set || !c->gates_set) return fail(DWKV_E_STATE, "basis and gates must be set before append");
  if (c->poisoned) return fail(DWKV_E_STATE, kPoisonMsg);
  PoisonGuard guard(c);
  int64_t total = 0, need = 0;
  if (c->seq_stamp.size() != (size_t)c->cfg.max_seqs) c->seq_stamp.assign(c->cfg.max_seqs, 0u);
  if (++c->stamp_gen == 0) { std::fill(c->seq_stamp.begin(), c->seq_stamp.end(), 0u); c->stamp_gen = 1; }
  for (int i = 0; i < n_seqs; ++i) {
    if (check_seq(c, seq_ids[i])) return fail(DWKV_E_INVALID, "bad sequence id");
    if (c->seq_stamp[seq_ids[i]] == c->stamp_gen) return fail(DWKV_E_INVALID, "duplicate sequence id");
    c->seq_stamp[seq_ids[i]] = c->stamp_gen;
    if (n_new[i] < 0) return fail(DWKV_E_INVALID, "negative n_new");
    if (n_new[i] > 0 && (!tier || !flag)) return fail(DWKV_E_INVALID, "NULL tier/flag");
    int rc = route_check(c, seq_ids[i], n_new[i], tier + total, flag + total, &need);
    if (rc) return rc;
    total += n_new[i];
  }
  if (total == 0) return DWKV_OK;
  if (!k_new || !v_new) return fail(DWKV_E_INVALID, "NULL k_new / v_new");
  if (need > (int64_t)c->free_pages.size()) return fail(DWKV_E_CAPACITY, "arena pages exhausted");
  if (total > 0x7fffffff) return fail(DWKV_E_INVALID, "too many tokens in one call");
  cudaStream_t st = (cudaStream_t)stream;
  // Large (prefill-sized) calls go in chunks of kChunk tokens of the call's row order: the host routes chunk i + 1 while the GPU
  // compresses chunk i. Rows keep their global index (TokDst::src), so every launch reads k_new / v_new in place.
  // (the first chunk is short, so that the GPU starts while the host still routes)
  constexpr int64_t kChunk = 16384, kFirst = 4096;
  std::vector<TokDst> dst, sorted;
  std::vector<int32_t> new_pages;
  int ridx = 0;
  for (int64_t g0 = 0, g1 = 0; g0 < total; g0 = g1) {
    g1 = std::min(total, g0 + ((g0 == 0 && total > kChunk) ? kFirst : kChunk));
    dst.clear();
    new_pages.clear();
    int64_t off = 0;
    for (int i = 0; i < n_seqs; ++i) {
      const int64_t lo = std::max(off, g0), hi = std::min(off + n_new[i], g1);
      if (lo < hi) {
        const size_t first = dst.size();
        guard.arm();
        route_commit(c, seq_ids[i], (int32_t)(hi - lo), tier + lo, flag + lo, &ridx, &dst, &new_pages);
        for (size_t k = first; k < dst.size(); ++k) dst[k].src = (int32_t)(lo + (int64_t)(k - first));
      }
      off += n_new[i];
    }
    // flagged tokens first, then by descending rank: only the flagged 16-token tiles run the reconstruction + int4 quantiser
    // part of the kernel, and a tile multiplies only the rank chunks its tokens keep. Counting sort, stable.
    {
      size_t start[8] = {0}, cnt[8] = {0};
      auto key = [](const TokDst& t) { return ((t.cls & 1) << 2) | (t.cls >> 1); };
      for (const TokDst& t : dst) cnt[key(t)]++;
      size_t acc = 0;
      for (int k = 7; k >= 0; --k) { start[k] = acc; acc += cnt[k]; }
      sorted.resize(dst.size());
      for (const TokDst& t : dst) sorted[start[key(t)]++] = t;
      dst.swap(sorted);
    }
    CompressRuns runs = {};
    for (size_t t0 = 0; t0 < dst.size(); t0 += 16) {            // the first token of a tile has its largest key
      const int cost = compress_tile_cost(dst[t0].cls & 1, c->geom.tier_rank[dst[t0].cls >> 1] / 8);
      if (runs.n == 0 || runs.cost[runs.n - 1] != cost) { runs.n++; runs.cost[runs.n - 1] = cost; runs.count[runs.n - 1] = 0; }
      runs.count[runs.n - 1]++;
      runs.per_lh += cost;
    }
    int rc = upload(c, c->tokdst_dev, dst.data(), dst.size() * sizeof(TokDst), st);
    if (rc) return rc;
    if (c->opt_time_scan && g0 == 0) {       // "compress_ms": from the first kernel of the call to the end of the last
      if (!c->ev_app0) { CU_OK(cudaEventCreate(&c->ev_app0)); CU_OK(cudaEventCreate(&c->ev_app1)); }
      CU_OK(cudaEventRecord(c->ev_app0, st));
    }
    c->launches += launch_compress_mma(c->arena, c->geom, (const TokDst*)c->tokdst_dev.p, (int)dst.size(), runs, (const __nv_bfloat16*)k_new,
                                       (const __nv_bfloat16*)v_new, c->BK, c->BV, c->gK, c->gV, c->n_sms, st);
  }
  if (c->opt_time_scan) { CU_OK(cudaEventRecord(c->ev_app1, st)); c->app_timed = true; }
  CU_OK(cudaGetLastError());
  guard.disarm();
  return DWKV_OK;
}

int dwkv_append_raw(dwkv_cache* c, int32_t seq_id, int32_t n, const uint8_t* tier, const uint8_t* flag,
                    const dwkv_raw_tokens* data, void* stream) {
  if (!c || n < 0) return fail(DWKV_E_INVALID, "NULL cache or negative n");
  if (check_seq(c, seq_id)) return fail(DWKV_E_INVALID, "bad sequence id");
  if (!c->basis_set || !c->gates_set) return fail(DWKV_E_STATE, "basis and gates must be set before append");
  if (c->poisoned) return fail(DWKV_E_STATE, kPoisonMsg);
  if (n == 0) return DWKV_OK;
  if (!tier || !flag || !data || !data->coefK || !data->coefV) return fail(DWKV_E_INVALID, "NULL argument");
  int64_t need = 0;
  int rc = route_check(c, seq_id, n, tier, flag, &need);
  if (rc) return rc;
  if (need > (int64_t)c->free_pages.size()) return fail(DWKV_E_CAPACITY, "arena pages exhausted");
  bool any_flag = false;
  for (int i = 0; i < n; ++i) any_flag |= flag[i] != 0;
  if (any_flag) {
    const bool modeA = data->residK && data->residV;
    const bool modeB = data->codeK && data->codeV && data->scaleK && data->scaleV;
    if (modeA == modeB) return fail(DWKV_E_INVALID, "exactly one residual mode (fp32 residuals, or codes + scales) must be given");
  }
  cudaStream_t st = (cudaStream_t)stream;
  std::vector<TokDst> dst;
  dst.reserve(n);
  std::vector<int32_t> new_pages;
  int ridx = 0;
  PoisonGuard guard(c);
  guard.arm();
  route_commit(c, seq_id, n, tier, flag, &ridx, &dst, &new_pages);
  rc = upload(c, c->tokdst_dev, dst.data(), dst.size() * sizeof(TokDst), st);
  if (rc) return rc;
  const bool modeA = data->residK && data->residV;
  c->launches += launch_scatter_raw(c->arena, c->geom, (const TokDst*)c->tokdst_dev.p, n, (const __nv_bfloat16*)data->coefK,
                                    (const __nv_bfloat16*)data->coefV, modeA ? data->residK : nullptr,
                                    modeA ? data->residV : nullptr, modeA ? nullptr : data->codeK, modeA ? nullptr : data->codeV,
                                    modeA ? nullptr : (const __half*)data->scaleK, modeA ? nullptr : (const __half*)data->scaleV, st);
  CU_OK(cudaGetLastError());
  guard.disarm();
  return DWKV_OK;
}

int dwkv_export_tokens(dwkv_cache* c, int32_t seq_id, int64_t t0, int64_t n, const dwkv_token_dump* out, void* stream) {
  if (!c || !out) return fail(DWKV_E_INVALID, "NULL argument");
  if (check_seq(c, seq_id)) return fail(DWKV_E_INVALID, "bad sequence id");
  const SeqState& S = c->seqs[seq_id];
  if (t0 < 0 || n < 0 || t0 + n > (int64_t)S.tier.size() || n > 0x7fffffff) return fail(DWKV_E_INVALID, "token range out of bounds");
  if (n == 0) return DWKV_OK;
  cudaStream_t st = (cudaStream_t)stream;
  std::vector<TokDst> dst;
  stored_token_table(c, S, t0, n, &dst);
  int rc = upload(c, c->tokdst_dev, dst.data(), dst.size() * sizeof(TokDst), st);
  if (rc) return rc;
  DumpPtrs o;
  o.coefK = (__nv_bfloat16*)out->coefK; o.coefV = (__nv_bfloat16*)out->coefV;
  o.codeK = out->codeK; o.codeV = out->codeV;
  o.scaleK = (__half*)out->scaleK; o.scaleV = (__half*)out->scaleV;
  o.deqK = out->deqK; o.deqV = out->deqV;
  c->launches += launch_gather(c->arena, c->geom, (const TokDst*)c->tokdst_dev.p, (int)n, o, st);
  CU_OK(cudaGetLastError());
  if (out->tier) CU_OK(cudaMemcpyAsync(out->tier, S.tier.data() + t0, n, cudaMemcpyHostToDevice, st));
  if (out->flag) CU_OK(cudaMemcpyAsync(out->flag, S.flag.data() + t0, n, cudaMemcpyHostToDevice, st));
  if (out->slot) CU_OK(cudaMemcpyAsync(out->slot, S.slot.data() + t0, n * sizeof(int32_t), cudaMemcpyHostToDevice, st));
  CU_OK(cudaStreamSynchronize(st));
  return DWKV_OK;
}

int dwkv_reset_seq(dwkv_cache* c, int32_t seq_id) {
  if (!c) return fail(DWKV_E_INVALID, "NULL cache");
  if (check_seq(c, seq_id)) return fail(DWKV_E_INVALID, "bad sequence id");
  cudaSetDevice(c->cfg.device);
  cudaDeviceSynchronize();     // pages may still be read by kernels in flight
  SeqState& S = c->seqs[seq_id];
  c->total_tokens -= (int64_t)S.tier.size();
  std::vector<int32_t> returned;
  for (int k = 0; k < kMaxClasses; ++k) {
    for (auto it = S.pages[k].rbegin(); it != S.pages[k].rend(); ++it) { c->free_pages.push_back(*it); returned.push_back(*it); }
    S.pages[k].clear();
    S.count[k] = 0;
  }
  if (!returned.empty()) {     // pages go back to the pool cleared; nothing may be in flight on them, before or after
    int rc = zero_pages(c, returned, 0);
    if (rc) { c->poisoned = true; return rc; }
    CU_OK(cudaDeviceSynchronize());
  }
  S.tier.clear(); S.flag.clear(); S.slot.clear();
  S.tok_dev_n = 0;
  c->version++;
  return DWKV_OK;
}

int dwkv_retier_seq(dwkv_cache* c, int32_t seq_id, const uint8_t* new_tier, const uint8_t* new_flag, void* stream) {
  if (!c || !new_tier || !new_flag) return fail(DWKV_E_INVALID, "NULL argument");
  if (check_seq(c, seq_id)) return fail(DWKV_E_INVALID, "bad sequence id");
  if (c->poisoned) return fail(DWKV_E_STATE, kPoisonMsg);
  cudaSetDevice(c->cfg.device);
  SeqState& S = c->seqs[seq_id];
  const int64_t n = (int64_t)S.tier.size();
  if (n == 0) return DWKV_OK;
  if (n > 0x7fffffff) return fail(DWKV_E_INVALID, "too many tokens");
  bool same = true;
  int64_t add[kMaxClasses] = {0, 0, 0, 0, 0, 0, 0, 0};
  for (int64_t i = 0; i < n; ++i) {
    if (new_tier[i] > S.tier[i] || new_flag[i] > S.flag[i])
      return fail(DWKV_E_INVALID, "re-tiering only lowers a token: new_tier <= tier and new_flag <= flag (the original vector is gone)");
    same = same && new_tier[i] == S.tier[i] && new_flag[i] == S.flag[i];
    add[2 * new_tier[i] + new_flag[i]]++;
  }
  if (same) return DWKV_OK;
  int64_t need = 0;
  for (int k = 0; k < c->n_classes; ++k) need += (add[k] + c->cl[k].tokens_per_page - 1) / c->cl[k].tokens_per_page;
  if (need > (int64_t)c->free_pages.size())      // the old pages are released only after the move
    return fail(DWKV_E_CAPACITY, "re-tiering needs " + std::to_string(need) + " free pages for the new layout, " +
                                     std::to_string(c->free_pages.size()) + " are free");
  cudaStream_t st = (cudaStream_t)stream;
  const CacheGeom& g = c->geom;
  const size_t LH = (size_t)g.L * g.H;
  const int64_t kChunkTok = 1024;
  const size_t per_tok = LH * ((size_t)g.r * 2 * 2 + (size_t)(g.d / 2) * 2 + (size_t)(g.d / 16) * 2 * 2);
  CU_OK(c->retier_ws.reserve((size_t)std::min<int64_t>(n, kChunkTok) * per_tok));
  CU_OK(c->tokdst_dev.reserve((size_t)std::min<int64_t>(n, kChunkTok) * sizeof(TokDst)));

  PoisonGuard guard(c);
  guard.arm();
  SeqState old = std::move(S);
  S = SeqState();
  S.tok_dev = old.tok_dev;          // the device token table's block moves to the new state; its entries are rebuilt by the next probe
  old.tok_dev = DevBuf();
  c->total_tokens -= n;
  std::vector<TokDst> dst_new, dst_old;
  std::vector<int32_t> new_pages;
  int ridx = 0;
  route_commit(c, seq_id, (int32_t)n, new_tier, new_flag, &ridx, &dst_new, &new_pages);
  for (int64_t t0 = 0; t0 < n; t0 += kChunkTok) {
    const int64_t m = std::min(kChunkTok, n - t0);
    uint8_t* w = (uint8_t*)c->retier_ws.p;
    DumpPtrs o;
    o.coefK = (__nv_bfloat16*)w; w += (size_t)m * LH * g.r * 2;
    o.coefV = (__nv_bfloat16*)w; w += (size_t)m * LH * g.r * 2;
    o.codeK = w; w += (size_t)m * LH * (g.d / 2);
    o.codeV = w; w += (size_t)m * LH * (g.d / 2);
    o.scaleK = (__half*)w; w += (size_t)m * LH * (g.d / 16) * 2;
    o.scaleV = (__half*)w;
    o.deqK = o.deqV = nullptr;
    stored_token_table(c, old, t0, m, &dst_old);
    int rc = upload(c, c->tokdst_dev, dst_old.data(), dst_old.size() * sizeof(TokDst), st);
    if (rc) return rc;
    c->launches += launch_gather(c->arena, g, (const TokDst*)c->tokdst_dev.p, (int)m, o, st);
    for (int64_t i = 0; i < m; ++i) dst_new[(size_t)(t0 + i)].ridx = new_flag[t0 + i] ? (int32_t)i : -1;    // row of the chunk's dump
    rc = upload(c, c->tokdst_dev, dst_new.data() + t0, (size_t)m * sizeof(TokDst), st);
    if (rc) return rc;
    c->launches += launch_scatter_raw(c->arena, g, (const TokDst*)c->tokdst_dev.p, (int)m, o.coefK, o.coefV, nullptr, nullptr, o.codeK,
                                      o.codeV, o.scaleK, o.scaleV, st);
    CU_OK(cudaGetLastError());
  }
  // the old pages go back to the pool, cleared, in stream order behind the reads above
  std::vector<int32_t> returned;
  for (int k = 0; k < kMaxClasses; ++k)
    for (auto it = old.pages[k].rbegin(); it != old.pages[k].rend(); ++it) returned.push_back(*it);
  int rc = zero_pages(c, returned, st);
  if (rc) return rc;
  for (int32_t pg : returned) c->free_pages.push_back(pg);
  c->version++;
  guard.disarm();
  return DWKV_OK;
}

int64_t dwkv_seq_len(const dwkv_cache* c, int32_t seq_id) {
  if (!c) return fail(DWKV_E_INVALID, "NULL cache");
  if (check_seq(c, seq_id)) return fail(DWKV_E_INVALID, "bad sequence id");
  return (int64_t)c->seqs[seq_id].tier.size();
}

int dwkv_footprint(const dwkv_cache* c, uint64_t* used_bytes, uint64_t* reserved_bytes, uint64_t* dense_equiv_bytes) {
  if (!c) return fail(DWKV_E_INVALID, "NULL cache");
  uint64_t used = 0;
  const uint64_t LH = (uint64_t)c->geom.L * c->geom.H, d = c->geom.d;
  for (const SeqState& S : c->seqs)
    for (int k = 0; k < c->n_classes; ++k)
      used += (uint64_t)S.count[k] * ((c->geom.i8 ? 2ull * (c->geom.tier_rank[k >> 1] + (c->geom.tier_rank[k >> 1] + 31) / 32) : 4ull * c->geom.tier_rank[k >> 1]) +
                                      (k & 1) * 2ull * (d / 2 + d / 8));
  if (used_bytes) *used_bytes = used * LH;
  if (reserved_bytes) *reserved_bytes = (uint64_t)pages_in_use(c) * c->page_bytes;
  if (dense_equiv_bytes) *dense_equiv_bytes = (uint64_t)c->total_tokens * LH * 4ull * d;
  return DWKV_OK;
}

int dwkv_set_option(dwkv_cache* c, const char* key, int64_t value) {
  if (!c || !key) return fail(DWKV_E_INVALID, "NULL argument");
  if (!strcmp(key, "max_unit_blocks")) c->opt_max_unit_blocks = value;
  else if (!strcmp(key, "time_scan")) { c->opt_time_scan = value; c->scan_samples = 0; }
  else if (!strcmp(key, "combine_warps")) c->opt_combine_warps = value;
  else if (!strcmp(key, "sketch_umma")) c->opt_sketch_umma = value;
  else if (!strcmp(key, "n_slices")) c->opt_n_slices = value;
  else if (!strcmp(key, "flag_cost_pct")) c->opt_flag_cost_pct = value;
  else if (!strcmp(key, "interleave")) c->opt_interleave = value;
  else if (!strcmp(key, "stamps_ptr")) c->opt_stamps_ptr = value;
  else if (!strcmp(key, "cost_coef_pct")) c->opt_cost_coef_pct = value;
  else if (!strcmp(key, "cost_tok")) c->opt_cost_tok = value;
  else if (!strcmp(key, "cost_seg")) c->opt_cost_seg = std::max<int64_t>(0, value);
  else if (!strcmp(key, "cost_resid_pct")) c->opt_cost_resid_pct = value;
  else if (!strcmp(key, "unit_kb")) c->opt_unit_kb = std::max<int64_t>(1, value);
  else if (!strcmp(key, "coef_int8")) {
    // storage format of the coefficient planes: fixed once tokens exist, like the basis (A19)
    if (value != 0 && value != 1) return fail(DWKV_E_INVALID, "coef_int8 must be 0 or 1");
    if (c->total_tokens != 0 || pages_in_use(c) != 0) return fail(DWKV_E_STATE, "coef_int8 cannot change while the cache holds tokens");
    c->geom.i8 = (int32_t)value;
    for (int k = 0; k < c->n_classes; ++k) c->cl[k] = make_class_layout(c->cfg.tier_rank[k >> 1], k & 1, c->cfg.d_head, c->geom.i8);
  }
  else return fail(DWKV_E_INVALID, std::string("unknown option ") + key);
  c->version++;
  c->opt_epoch++;
  return DWKV_OK;
}

int64_t dwkv_launch_count(const dwkv_cache* c) { return c ? c->launches : 0; }

double dwkv_get_stat(dwkv_cache* c, const char* key) {
  if (!c || !key) return -1.0;
  if (!strcmp(key, "plan_slices")) return c->plan3.valid ? (double)c->plan3.n_slices : -1.0;     // of the last decode call
  if (!strcmp(key, "plan_slots")) return c->plan3.valid ? (double)c->plan3.n_slots : -1.0;
  if (!strcmp(key, "plan_segments")) return c->plan3.valid ? (double)c->plan3.n_segs : -1.0;
  if (!strcmp(key, "scan_samples")) return (double)(c->scan_samples < dwkv_cache::kScanRing ? c->scan_samples : dwkv_cache::kScanRing);
  if (!strncmp(key, "scan_ms@", 8)) {                  // "scan_ms@i": sample i (0 = oldest kept) of the calls timed since "time_scan" was set
    const int64_t n = c->scan_samples < dwkv_cache::kScanRing ? c->scan_samples : dwkv_cache::kScanRing;
    const int64_t k = atoll(key + 8);
    if (k < 0 || k >= n) return -1.0;
    const int i = (int)((c->scan_samples - n + k) % dwkv_cache::kScanRing);
    if (cudaEventSynchronize(c->ev_scan1[i]) != cudaSuccess) return -1.0;
    float ms = -1.f;
    if (cudaEventElapsedTime(&ms, c->ev_scan0[i], c->ev_scan1[i]) != cudaSuccess) return -1.0;
    return (double)ms;
  }
  const bool s_mean = !strcmp(key, "scan_ms_mean"), s_min = !strcmp(key, "scan_ms_min");
  if (!strcmp(key, "scan_ms") || s_mean || s_min) {     // last kernel / mean / min over the (up to 64) kernels timed since "time_scan" was set
    if (c->scan_samples == 0) return -1.0;
    const int64_t n = c->scan_samples < dwkv_cache::kScanRing ? c->scan_samples : dwkv_cache::kScanRing;
    const int64_t first = (s_mean || s_min) ? c->scan_samples - n : c->scan_samples - 1;
    double sum = 0.0, mn = 1e30;
    for (int64_t k = first; k < c->scan_samples; ++k) {
      const int i = (int)(k % dwkv_cache::kScanRing);
      if (cudaEventSynchronize(c->ev_scan1[i]) != cudaSuccess) return -1.0;
      float ms = -1.f;
      if (cudaEventElapsedTime(&ms, c->ev_scan0[i], c->ev_scan1[i]) != cudaSuccess) return -1.0;
      sum += ms; mn = ms < mn ? ms : mn;
    }
    return s_min ? mn : sum / (double)(c->scan_samples - first);
  }
  if (!strcmp(key, "compress_ms")) {
    if (!c->app_timed) return -1.0;
    if (cudaEventSynchronize(c->ev_app1) != cudaSuccess) return -1.0;
    float ms = -1.f;
    if (cudaEventElapsedTime(&ms, c->ev_app0, c->ev_app1) != cudaSuccess) return -1.0;
    return (double)ms;
  }
  return -1.0;
}

}  // extern "C"

// =================================================================================================================
// decode: work-list planner + launch sequence
// =================================================================================================================
namespace {

// Plan of the fused persistent kernel. Linear order of the step's work: (sequence b, lh = layer * H + head, unit of b,
// sub-block); a unit is one page stripe of a (sequence, class). The order is cut into n_slices contiguous slices of equal
// COST (bytes, flagged bytes weighted by opt_flag_cost_pct) at sub-block granularity, one per warp. A slice touches one or a
// few segments (b, lh); every (slice, segment) contact yields one partial, numbered contiguously per segment (pstart).
// Depends on the sequence set, the token counts, the layer count and the options only.
int build_plan3(dwkv_cache* c, int32_t n_seqs, const int32_t* seq_ids, int n_lsel, cudaStream_t st) {
  Plan3& P = c->plan3;
  if (P.valid && P.version == c->version && P.n_lsel == n_lsel && (int)P.seq_ids.size() == n_seqs &&
      std::equal(P.seq_ids.begin(), P.seq_ids.end(), seq_ids))
    return DWKV_OK;
  // (the fast path below keeps the old slice cut: only under the same planner options)
  const bool same_call = P.valid && P.n_lsel == n_lsel && P.opt_epoch == c->opt_epoch && (int)P.seq_ids.size() == n_seqs &&
                         std::equal(P.seq_ids.begin(), P.seq_ids.end(), seq_ids);
  P.valid = false;
  const int LH = n_lsel * c->geom.H;
  const double flag_w = (double)c->opt_flag_cost_pct / 100.0;
  const double seg_ovh = (double)c->opt_cost_seg;
  // class order inside a sequence: interleaved, every slice sees the sequence's class mix and the cost model drops out of the
  // balance; measured -1.2 % at G = 8 (70B shape) and -1.7 % on a single sequence, neutral (+-0.3 %) on batches at G = 4
  // (re-measured at the end of round 2 on per-layer calls: -2 % at batch 2, -4 % at batch 4, +2 % at batch 8; all-layer -0.3 % throughout)
  const bool interleave = c->opt_interleave >= 0 ? c->opt_interleave != 0 : (c->geom.G > 4 || n_seqs <= 4);
  // per-token and per-residual-byte work grows with the query heads per kv head (fits at G = 4: 24 / 235 %, G = 8: 48 / 265 %)
  const double cost_tok = c->opt_cost_tok >= 0 ? (double)c->opt_cost_tok : 6.0 * c->geom.G;
  const double cost_resid_pct = c->opt_cost_resid_pct >= 0 ? (double)c->opt_cost_resid_pct : 205.0 + 7.5 * c->geom.G;
  std::vector<Unit> units;
  std::vector<int32_t> ustart(n_seqs + 1, 0), unsub;
  std::vector<double> upre, usub, seq_cost(n_seqs, 0.0), cumB(n_seqs + 1, 0.0);
  for (int b = 0; b < n_seqs; ++b) {
    ustart[b] = (int32_t)units.size();
    const SeqState& S = c->seqs[seq_ids[b]];
    double acc = 0.0;
    // units of ~opt_unit_kb per class, then the classes are interleaved in proportion (largest remainder) so that every
    // slice of the order sees the sequence's class mix: classes differ in instructions per byte, equal-cost slices of one
    // class each would finish at different times
    struct CU { Unit u; double cost_sub; int nsub; };
    std::vector<CU> byc[kMaxClasses];
    for (int fl = 1; fl >= 0; --fl) {
      for (int tr = c->cfg.n_tiers - 1; tr >= 0; --tr) {
        const int k = 2 * tr + fl;
        if (S.count[k] == 0) continue;
        const ClassLayout& cl = c->cl[k];
        const int64_t tpp = cl.tokens_per_page;
        int64_t ub = c->opt_max_unit_blocks > 0 ? c->opt_max_unit_blocks
                                                : std::max<int64_t>(1, (c->opt_unit_kb * 1024 + cl.block_bytes / 2) / cl.block_bytes);
        ub = std::min<int64_t>(ub, cl.blocks_per_page);
        // cost of a sub-block in byte-equivalents: the warp is partly issue bound, so tokens (softmax work) and residual
        // bytes (int4 unpack, group scales) weigh more than coefficient bytes (fit to per-warp finish times)
        // (8-bit coefficient planes: half the bytes per coefficient and ~1.5x the instructions -- the codes are widened in
        //  registers -- so a coefficient byte weighs 3x; measured optimum on the 64K batch-8 and the ragged workload)
        const double cost_sub = 0.01 * (double)c->opt_cost_coef_pct * (c->geom.i8 ? 3.0 : 1.0) * 2.0 * cl.coef_bytes + cost_tok * cl.sub_tok +
                                0.01 * cost_resid_pct * flag_w * 2.0 * (cl.code_bytes + cl.scale_bytes);
        for (size_t pi = 0; pi < S.pages[k].size(); ++pi) {
          const int64_t tok_in_page = std::min<int64_t>(tpp, S.count[k] - (int64_t)pi * tpp);
          if (tok_in_page <= 0) break;
          const int64_t nblk = (tok_in_page + kBlockTok - 1) / kBlockTok;
          for (int64_t b0 = 0; b0 < nblk; b0 += ub) {
            CU x;
            Unit& u = x.u;
            u.page_off = (int64_t)S.pages[k][pi] * (int64_t)c->page_bytes;
            u.blk0 = (int32_t)b0;
            u.nblk = (int32_t)std::min<int64_t>(ub, nblk - b0);
            u.ntok = (int32_t)(std::min<int64_t>(tok_in_page, (b0 + u.nblk) * kBlockTok) - b0 * kBlockTok);
            u.cls = (int16_t)k;
            u.b = (int16_t)b;
            u.epart = -1;
            u.rk = c->geom.tier_rank[tr];
            x.cost_sub = cost_sub;
            x.nsub = (u.ntok + cl.sub_tok - 1) / cl.sub_tok;
            byc[k].push_back(x);
          }
        }
      }
    }
    size_t taken[kMaxClasses] = {0, 0, 0, 0, 0, 0, 0, 0}, left = 0;
    for (int k = 0; k < kMaxClasses; ++k) left += byc[k].size();
    while (left > 0) {
      int best = -1;
      double best_key = 0.0;
      for (int k = 0; k < kMaxClasses; ++k) {
        if (taken[k] == byc[k].size()) continue;
        const double key = interleave ? ((double)taken[k] + 0.5) / (double)byc[k].size() : (double)((k & 1) ? 0 : 8) + (7 - k);
        if (best < 0 || key < best_key) { best = k; best_key = key; }
      }
      const CU& x = byc[best][taken[best]++];
      units.push_back(x.u);
      upre.push_back(acc);
      usub.push_back(x.cost_sub);
      unsub.push_back(x.nsub);
      acc += (double)x.nsub * x.cost_sub;
      --left;
    }
    seq_cost[b] = acc + seg_ovh;       // entering a segment costs a prologue (q pre-projection) and a partial flush
    cumB[b + 1] = cumB[b] + seq_cost[b] * LH;
  }
  ustart[n_seqs] = (int32_t)units.size();
  if (same_call && units.size() == P.units.size() && unsub == P.unsub) {
    // fast path (the common decode step: a few tokens appended inside existing sub-blocks): same units up to their token counts
    bool same = true;
    for (size_t i = 0; i < units.size() && same; ++i) {
      const Unit &a = units[i], &b = P.units[i];
      same = a.page_off == b.page_off && a.blk0 == b.blk0 && a.nblk == b.nblk && a.cls == b.cls && a.b == b.b && a.rk == b.rk;
    }
    if (same) {
      int rc = upload(c, c->plan3_dev, units.data(), units.size() * sizeof(Unit), st);     // the unit array is the head of the blob
      if (rc) return rc;
      P.units.swap(units);
      P.version = c->version;
      P.valid = true;
      return DWKV_OK;
    }
  }
  const int n_units = (int)units.size(), S_total = n_seqs * LH;
  const int Wmax = scan3_num_slices(c->n_sms);
  const double C = cumB[n_seqs];
  // small calls (one layer of one 64K sequence: 33 MB) are latency bound: with one slice per warp a warp streams < 30 KB and
  // every segment collects ~150 partials; fewer, longer slices (~85 K cost units = ~55 KB each, the same number of warps on
  // every SM) shorten both the scan and the combine (measured: 707 -> 635 us per 32 per-layer calls at batch 1)
  int W = Wmax;
  if (c->opt_n_slices > 0) W = (int)std::min<int64_t>(c->opt_n_slices, Wmax);
  else if (C >= 8e6 && C < 50e3 * (double)Wmax && Wmax % c->n_sms == 0) {      // (below ~6 MB everything is launch latency)
    const int per_sm = std::min(Wmax / c->n_sms, std::max(2, (int)std::floor(C / (85e3 * (double)c->n_sms) + 0.5)));
    W = per_sm * c->n_sms;
  }
  const int NSL = W;
  struct Pos { int32_t seg, u, sub; };
  auto less = [](const Pos& a, const Pos& b) { return a.seg != b.seg ? a.seg < b.seg : (a.u != b.u ? a.u < b.u : a.sub < b.sub); };
  std::vector<Pos> pos(NSL + 1);
  const Pos end_pos{S_total, n_units, 0};
  for (int k = 0; k <= NSL; ++k) {
    Pos q = end_pos;
    if (k < NSL) {
      const double target = C * (double)k / (double)W;
      int b = (int)(std::upper_bound(cumB.begin(), cumB.end(), target) - cumB.begin()) - 1;
      b = std::min(std::max(b, 0), n_seqs - 1);
      double rem = target - cumB[b];
      int lh = std::min(LH - 1, (int)std::floor(rem / seq_cost[b]));
      rem -= (double)lh * seq_cost[b];
      rem = std::max(0.0, rem - seg_ovh);   // the overhead sits at the start of the segment
      int u = (int)(std::upper_bound(upre.begin() + ustart[b], upre.begin() + ustart[b + 1], rem) - upre.begin()) - 1;
      u = std::min(std::max(u, ustart[b]), ustart[b + 1] - 1);
      int sub = (int)std::floor((rem - upre[u]) / usub[u] + 0.5);
      sub = std::max(sub, 0);
      if (sub >= unsub[u]) {          // normalise: a position never points past the last sub-block of a unit
        sub = 0;
        if (++u == ustart[b + 1]) {
          if (++lh == LH) { lh = 0; ++b; }
          u = b < n_seqs ? ustart[b] : n_units;
        }
      }
      q = b < n_seqs ? Pos{b * LH + lh, u, sub} : end_pos;
    }
    if (k > 0 && less(q, pos[k - 1])) q = pos[k - 1];
    pos[k] = q;
  }
  pos[0] = Pos{0, 0, 0};
  // partial slots: contacts (slice, segment), numbered per segment in slice order
  std::vector<int32_t> pstart(S_total + 1, 0), seen(S_total, 0);
  auto last_seg = [&](const Pos& e) {
    if (e.seg >= S_total) return S_total - 1;
    const int b = e.seg / LH;
    return (e.u == ustart[b] && e.sub == 0) ? e.seg - 1 : e.seg;
  };
  std::vector<int32_t> wentry(4 * (size_t)(NSL + 1), 0);
  for (int w = 0; w <= NSL; ++w) {
    wentry[4 * w + 0] = pos[w].seg; wentry[4 * w + 1] = pos[w].u; wentry[4 * w + 2] = pos[w].sub; wentry[4 * w + 3] = 0;
  }
  for (int w = 0; w < NSL; ++w) {
    if (!less(pos[w], pos[w + 1])) continue;
    for (int s = pos[w].seg, s1 = last_seg(pos[w + 1]); s <= s1; ++s) pstart[s + 1]++;
  }
  for (int s = 0; s < S_total; ++s) pstart[s + 1] += pstart[s];
  for (int w = 0; w < NSL; ++w) {
    if (!less(pos[w], pos[w + 1])) continue;
    wentry[4 * w + 3] = pstart[pos[w].seg] + seen[pos[w].seg];
    for (int s = pos[w].seg, s1 = last_seg(pos[w + 1]); s <= s1; ++s) seen[s]++;
  }
  // one blob: units | ustart | wentry | pstart
  const size_t sz_units = units.size() * sizeof(Unit);
  P.off_ustart = (sz_units + 15) & ~(size_t)15;
  P.off_wentry = (P.off_ustart + ustart.size() * sizeof(int32_t) + 15) & ~(size_t)15;
  P.off_pstart = (P.off_wentry + wentry.size() * sizeof(int32_t) + 15) & ~(size_t)15;
  const size_t total = P.off_pstart + pstart.size() * sizeof(int32_t);
  std::vector<uint8_t> blob(total, 0);
  memcpy(blob.data(), units.data(), sz_units);
  memcpy(blob.data() + P.off_ustart, ustart.data(), ustart.size() * sizeof(int32_t));
  memcpy(blob.data() + P.off_wentry, wentry.data(), wentry.size() * sizeof(int32_t));
  memcpy(blob.data() + P.off_pstart, pstart.data(), pstart.size() * sizeof(int32_t));
  int rc = upload(c, c->plan3_dev, blob.data(), total, st);
  if (rc) return rc;
  P.n_units = n_units; P.n_slices = NSL; P.n_segs = S_total; P.n_slots = pstart[S_total];
  P.units.swap(units);
  P.unsub.swap(unsub);
  P.seq_ids.assign(seq_ids, seq_ids + n_seqs);
  P.n_lsel = n_lsel;
  P.opt_epoch = c->opt_epoch;
  P.version = c->version;
  P.valid = true;
  return DWKV_OK;
}

int decode3(dwkv_cache* c, int32_t layer, int32_t n_seqs, const int32_t* seq_ids, const void* q, float* out, cudaStream_t st) {
  const CacheGeom& g = c->geom;
  const int Lsel = layer < 0 ? g.L : 1, layer0 = layer < 0 ? 0 : layer;
  // warp partials + a separate combine kernel, for all-layer and per-layer calls alike: the variants with the split-combine fused
  // into the decode kernel (last-arrival epilogue, CTA-level merge of the partials) were built, parity-tested and measured slower
  // (git history before this line's commit holds them)
  int rc = build_plan3(c, n_seqs, seq_ids, Lsel, st);
  if (rc) return rc;
  const Plan3& P = c->plan3;
  CU_OK(c->part.reserve((size_t)P.n_slots * g.G * (2 + g.r + g.d) * sizeof(float)));
  const uint8_t* blob = (const uint8_t*)c->plan3_dev.p;
  Scan3Params sp;
  sp.arena = c->arena;
  sp.units = (const Unit*)blob;
  sp.ustart = (const int32_t*)(blob + P.off_ustart);
  sp.wentry = (const int4*)(blob + P.off_wentry);
  sp.pstart = (const int32_t*)(blob + P.off_pstart);
  sp.q = (const __nv_bfloat16*)q; sp.BK = c->BK; sp.gK = c->gK;
  sp.part = (float*)c->part.p;
  sp.stamps = (unsigned long long*)c->opt_stamps_ptr;
  sp.n_slices = P.n_slices; sp.n_segs = P.n_segs;
  sp.layer0 = layer0; sp.Lq = Lsel; sp.LH = Lsel * g.H; sp.w = g.w;
  sp.H = g.H; sp.G = g.G; sp.r = g.r; sp.d = g.d;
  sp.cscale = c->softmax_scale * 1.4426950408889634f;
  sp.zero = 0.f;
  sp.i8 = g.i8;
  sp.rot = (n_seqs == 1 && Lsel > 1) ? 53 : 0;
  const int ev_i = (int)(c->scan_samples % dwkv_cache::kScanRing);
  if (c->opt_time_scan) {
    if (!c->ev_scan0[ev_i]) { CU_OK(cudaEventCreate(&c->ev_scan0[ev_i])); CU_OK(cudaEventCreate(&c->ev_scan1[ev_i])); }
    CU_OK(cudaEventRecord(c->ev_scan0[ev_i], st));
  }
  cudaError_t lerr = cudaSuccess;
  const int n = launch_scan3(sp, c->n_sms, st, &lerr);
  if (n == 0) return fail(DWKV_E_INVALID, "no fused decode kernel instance for this shape");
  CU_OK(lerr);
  c->launches += n;
  if (c->opt_time_scan) { CU_OK(cudaEventRecord(c->ev_scan1[ev_i], st)); ++c->scan_samples; }
  Combine3Params cp;
  cp.pstart = sp.pstart; cp.part = sp.part; cp.BV = c->BV; cp.gV = c->gV; cp.out = out;
  cp.layer0 = layer0; cp.Lq = Lsel; cp.LH = sp.LH; cp.w = g.w; cp.H = g.H; cp.G = g.G; cp.r = g.r; cp.d = g.d;
  // more than ~8 partials per segment (per-layer calls): the 4 warps of a CTA share one head's partial list; a 16-warp shape was
  // carried until the combine's dependent round trips were cut to two, after which it lost everywhere (per-layer step at batch 1:
  // 614 us against 582 us with 4 warps) and was removed
  const int split = (c->opt_combine_warps == 1 || c->opt_combine_warps == 4) ? (int)c->opt_combine_warps
                                                                             : (P.n_slots > 8LL * P.n_segs ? 4 : 1);
  c->launches += launch_combine3(cp, P.n_segs, split, st, &lerr);
  CU_OK(lerr);
  CU_OK(cudaGetLastError());
  return DWKV_OK;
}

}  // namespace

extern "C" int dwkv_decode_attention(dwkv_cache* c, int32_t layer, int32_t n_seqs, const int32_t* seq_ids, const void* q,
                                     float* out, void* stream) {
  if (!c || !seq_ids || !q || !out || n_seqs <= 0) return fail(DWKV_E_INVALID, "NULL argument or n_seqs <= 0");
  if (layer < -1 || layer >= c->geom.L) return fail(DWKV_E_INVALID, "layer out of range");
  if (!c->basis_set || !c->gates_set) return fail(DWKV_E_STATE, "basis and gates must be set before decode");
  if (c->poisoned) return fail(DWKV_E_STATE, kPoisonMsg);
  if (n_seqs > 32767) return fail(DWKV_E_INVALID, "too many sequences in one call");
  if (c->seq_stamp.size() != (size_t)c->cfg.max_seqs) c->seq_stamp.assign(c->cfg.max_seqs, 0u);
  if (++c->stamp_gen == 0) { std::fill(c->seq_stamp.begin(), c->seq_stamp.end(), 0u); c->stamp_gen = 1; }
  for (int i = 0; i < n_seqs; ++i) {
    if (check_seq(c, seq_ids[i])) return fail(DWKV_E_INVALID, "bad sequence id");
    if (c->seq_stamp[seq_ids[i]] == c->stamp_gen) return fail(DWKV_E_INVALID, "duplicate sequence id");
    c->seq_stamp[seq_ids[i]] = c->stamp_gen;
    if (c->seqs[seq_ids[i]].tier.empty()) return fail(DWKV_E_EMPTY, "decode on an empty sequence (reading A17)");
  }
  cudaStream_t st = (cudaStream_t)stream;
  return decode3(c, layer, n_seqs, seq_ids, q, out, st);
}

extern "C" int dwkv_probe_token_stats(dwkv_cache* c, int32_t layer, int32_t seq_id, const void* q, float* mass, float* spike, void* stream) {
  if (!c || !q || !mass || !spike) return fail(DWKV_E_INVALID, "NULL argument");
  if (layer < 0 || layer >= c->geom.L) return fail(DWKV_E_INVALID, "layer out of range");
  if (check_seq(c, seq_id)) return fail(DWKV_E_INVALID, "bad sequence id");
  if (!c->basis_set || !c->gates_set) return fail(DWKV_E_STATE, "basis and gates must be set before the probe");
  SeqState& S = c->seqs[seq_id];
  const int64_t T = (int64_t)S.tier.size();
  if (T == 0) return fail(DWKV_E_EMPTY, "token statistics of an empty sequence");
  if (T > 0x7fffffff) return fail(DWKV_E_INVALID, "sequence too long");
  cudaStream_t st = (cudaStream_t)stream;
  if (S.tok_dev_n < T) {        // bring the device-resident token table up to date: only the tokens appended since the last probe
    std::vector<TokDst> dst;
    stored_token_table(c, S, S.tok_dev_n, T - S.tok_dev_n, &dst);
    CU_OK(S.tok_dev.grow_keep((size_t)T * sizeof(TokDst), (size_t)S.tok_dev_n * sizeof(TokDst), st));
    int rc = upload_to(c, (uint8_t*)S.tok_dev.p + (size_t)S.tok_dev_n * sizeof(TokDst), dst.data(), dst.size() * sizeof(TokDst), st);
    if (rc) return rc;
    S.tok_dev_n = T;
  }
  CU_OK(c->probe_ws.reserve(token_stats_scratch_bytes(c->geom, T)));
  c->launches += launch_token_stats(c->arena, c->geom, (const TokDst*)S.tok_dev.p, (int)T, layer, (const __nv_bfloat16*)q, c->BK, c->gK,
                                    c->softmax_scale * 1.4426950408889634f, (float*)c->probe_ws.p, mass, spike, st);
  CU_OK(cudaGetLastError());
  return DWKV_OK;
}

extern "C" int dwkv_probe_error(dwkv_cache* c, int32_t layer, int32_t seq_id, int32_t n_q, const void* q, const void* K_ref,
                                const void* V_ref, float eps, float* e_out, void* stream) {
  if (!c || !q || !K_ref || !V_ref || !e_out || n_q <= 0) return fail(DWKV_E_INVALID, "NULL argument or n_q <= 0");
  if (layer < 0 || layer >= c->geom.L) return fail(DWKV_E_INVALID, "layer out of range");
  if (check_seq(c, seq_id)) return fail(DWKV_E_INVALID, "bad sequence id");
  if (!c->basis_set || !c->gates_set) return fail(DWKV_E_STATE, "basis and gates must be set before the probe");
  const int64_t T = (int64_t)c->seqs[seq_id].tier.size();
  if (T == 0) return fail(DWKV_E_EMPTY, "probe on an empty sequence");
  const CacheGeom& g = c->geom;
  const int Hq = g.H * g.G;
  cudaStream_t st = (cudaStream_t)stream;
  const size_t out_elems = (size_t)n_q * Hq * g.d;
  const size_t dense_ws = (size_t)dwkv_dense_workspace_bytes(1, 1, Hq, g.d, T);
  CU_OK(c->probe_ws.reserve(2 * out_elems * sizeof(float) + dense_ws));
  float* o_cmp = (float*)c->probe_ws.p;
  float* o_ref = o_cmp + out_elems;
  void* ws = (void*)(o_ref + out_elems);
  const __nv_bfloat16* qb = (const __nv_bfloat16*)q;
  for (int i = 0; i < n_q; ++i) {       // every probed position attends to all T cached tokens (reading A10)
    int rc = decode3(c, layer, 1, &seq_id, qb + (size_t)i * Hq * g.d, o_cmp + (size_t)i * Hq * g.d, st);
    if (rc) return rc;
    rc = dwkv_dense_decode_attention(K_ref, V_ref, qb + (size_t)i * Hq * g.d, o_ref + (size_t)i * Hq * g.d, ws, 1, 1, g.H, Hq, g.d, T,
                                     c->softmax_scale, stream);
    if (rc) return fail(rc, "dense reference attention failed");
    c->launches += 2;
  }
  c->launches += launch_probe_error(o_ref, o_cmp, e_out, n_q, g.H, g.G, g.d, eps, st);
  CU_OK(cudaGetLastError());
  return DWKV_OK;
}
