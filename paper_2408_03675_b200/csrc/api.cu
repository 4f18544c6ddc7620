// api.cu -- the C ABI of libnacl_evict.so (include/nacl_evict.h): argument validation, workspace
// carve-up and the launch sequence of one eviction call.
// Host code only enqueues; it never reads device memory and never synchronises (except
// nacl_evict_host, which is documented as synchronous).
#include <mutex>
#include <new>
#include <vector>

#include "nacl_internal.cuh"

namespace nacl {

static thread_local int g_last_cuda_error = 0;

static size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// ------------------------------------------------------------------ per-stage timing
struct ProfRecord { int stage; cudaEvent_t a, b; };
static std::mutex g_prof_mu;
static bool g_prof_on = false;
static std::vector<ProfRecord> g_prof_pending;
static std::vector<cudaEvent_t> g_prof_free;
static double g_prof_ms[ST_COUNT] = {};
static int64_t g_prof_n[ST_COUNT] = {};

static cudaEvent_t prof_event() {
  if (!g_prof_free.empty()) { cudaEvent_t e = g_prof_free.back(); g_prof_free.pop_back(); return e; }
  cudaEvent_t e = nullptr;
  if (cudaEventCreate(&e) != cudaSuccess) { cudaGetLastError(); return nullptr; }
  return e;
}

StageScope::StageScope(int stage, cudaStream_t st) : stage_(stage), st_(st), a_(nullptr), b_(nullptr) {
  std::lock_guard<std::mutex> lk(g_prof_mu);
  if (!g_prof_on) return;
  a_ = prof_event();
  b_ = prof_event();
  if (!a_ || !b_) {
    if (a_) g_prof_free.push_back(a_);
    if (b_) g_prof_free.push_back(b_);
    a_ = b_ = nullptr;
    return;
  }
  cudaEventRecord(a_, st);
}
StageScope::~StageScope() {
  if (!a_) return;
  // the pair enters the pending list only once both events are recorded: a nacl_profile_read in between never sees half a scope
  cudaEventRecord(b_, st_);
  std::lock_guard<std::mutex> lk(g_prof_mu);
  g_prof_pending.push_back(ProfRecord{stage_, a_, b_});
}

SplitPlan make_split_plan(int batch, int L, int Hkv) {
  // about 6 work items per SM (and per sweep) so that a dynamically scheduled grid ends with a short tail
  const long heads = (long)batch * Hkv;
  const long items_target = 6L * kNumSMs;
  long per_head = (items_target + heads - 1) / heads;
  if (per_head < 1) per_head = 1;
  long chunk = ((long)L + per_head - 1) / per_head;
  chunk = (chunk + 127) / 128 * 128;
  if (chunk < 128) chunk = 128;
  SplitPlan sp;
  sp.chunk = (int)chunk;
  sp.n_chunks = (int)(((long)L + chunk - 1) / chunk);
  return sp;
}

Workspace carve_workspace(void* base, int batch, int L, int Hq, int Hkv, int P) {
  const SplitPlan sp = make_split_plan(batch, L, Hkv);
  const size_t n_rows = (size_t)batch * Hq * P;
  const size_t n_imp = (size_t)batch * Hkv * L;
  size_t off = 0;
  char* b = static_cast<char*>(base);
  Workspace ws;
  // first, so that its place does not depend on the other sizes: evict_impl keeps track of how much of it is known to be zero
  ws.sync = reinterpret_cast<int*>(b + off);    off = align_up(off + sync_ints((size_t)batch * Hkv) * sizeof(int), 256);
  size_t n_part = n_rows * sp.n_chunks;  // generic path; the tensor-core path keeps one partial per (CTA + head, warpgroup, row)
  const size_t n_part_tc = score_tc_part_elems(batch * Hkv, (Hq / Hkv) * P);
  if (n_part_tc > n_part) n_part = n_part_tc;
  ws.part = reinterpret_cast<float2*>(b + off); off = align_up(off + n_part * sizeof(float2), 256);
  ws.lse = reinterpret_cast<float*>(b + off);   off = align_up(off + n_rows * sizeof(float), 256);
  ws.imp = reinterpret_cast<float*>(b + off);   off = align_up(off + n_imp * sizeof(float), 256);
  ws.key = reinterpret_cast<uint32_t*>(b + off); off = align_up(off + select_scratch_words(batch, Hkv, L) * sizeof(uint32_t), 256);
  ws.imp_sh = reinterpret_cast<float*>(b + off); off = align_up(off + (size_t)batch * L * sizeof(float), 256);
  ws.idx_sh = reinterpret_cast<int32_t*>(b + off); off = align_up(off + (size_t)batch * L * sizeof(int32_t), 256);
  ws.idx_tmp = reinterpret_cast<int32_t*>(b + off); off = align_up(off + n_imp * sizeof(int32_t), 256);
  ws.bytes = off;
  return ws;
}

// ------------------------------------------------------------------ validation
static int validate_shape(int dtype, int batch, int L, int Hq, int Hkv, int d, int P) {
  if (dtype != NACL_DTYPE_F32 && dtype != NACL_DTYPE_BF16) return NACL_ERR_UNSUPPORTED;
  if (batch < 1 || L < 1 || Hq < 1 || Hkv < 1 || d < 1 || P < 1) return NACL_ERR_SHAPE;
  if (Hq % Hkv != 0 || P > L || L > (1 << 24)) return NACL_ERR_SHAPE;
  if (d % 16 != 0 || d > 256) return NACL_ERR_SHAPE;
  if ((long)batch * Hkv > 65535 || batch > 65535) return NACL_ERR_SHAPE;
  if ((long)batch * Hq * P > (1L << 30)) return NACL_ERR_SHAPE;
  return NACL_OK;
}

static int validate_budget(int L, int budget_proxy, int budget_random, int n_sink, int n_recent, int n_protect = 0) {
  if (budget_proxy < 0 || budget_random < 0 || n_sink < 0 || n_recent < 0 || n_protect < 0) return NACL_ERR_BUDGET;
  const long n_prot = (long)n_sink + n_recent;
  if (n_prot > L) return NACL_ERR_BUDGET;
  if (budget_proxy < n_prot + n_protect) return NACL_ERR_BUDGET;  // protected tokens count inside budget_proxy (R7)
  if ((long)budget_proxy + budget_random > L) return NACL_ERR_BUDGET;
  return NACL_OK;
}

static bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

// ------------------------------------------------------------------ internal buffers
// The internal workspace is keyed by (device, stream): calls on one stream are ordered and may share scratch, calls on
// different streams may run at the same time and must not.  A buffer that is too small is replaced; the old one may
// still be in use by calls enqueued earlier, so it is RETIRED with the event that the last call using it recorded behind
// its last kernel, and freed by a later call once that event has completed.  At most kMaxStreamWorkspaces streams keep
// a workspace per device: beyond that the least recently used one is retired the same way (an application that creates
// and destroys streams does not accumulate them).  A workspace that was ever used while its stream was being captured
// may be referenced by a graph that is replayed at any later time: it is never freed before nacl_release.
constexpr size_t kMaxStreamWorkspaces = 16;
struct WsEntry {
  cudaStream_t stream;
  void* ptr;
  size_t bytes;
  size_t sync_clean;   // leading bytes known to be zero
  cudaEvent_t done;    // recorded behind the last kernel of the latest call that used ptr
  uint64_t last_use;   // DeviceCache::tick of that call
  bool captured;       // used under stream capture at least once
};
struct RetiredWs { void* ptr; cudaEvent_t done; };  // done == nullptr: keep until nacl_release
struct DeviceCache {
  std::vector<WsEntry> ws;
  std::vector<RetiredWs> retired;
  uint64_t tick = 0;
  void* stage[2][6] = {};         // nacl_evict_host(_batch): two staging slots of K V Q oK oV idx ...
  size_t stage_bytes[2][6] = {};
  cudaStream_t stream[2] = {nullptr, nullptr};  // ... with a stream each
  cudaStream_t bstream[2] = {nullptr, nullptr};  // nacl_evict_batch: the two streams the calls alternate on
  cudaEvent_t bfork = nullptr, bjoin[2] = {nullptr, nullptr};
};
static std::mutex g_mu;       // guards g_cache
static std::mutex g_host_mu;  // serialises nacl_evict_host (its staging buffers are shared per device)
static DeviceCache g_cache[64];

static cudaError_t grow(void** p, size_t* have, size_t want) {
  if (*have >= want && *p) return cudaSuccess;
  if (*p) {
    cudaError_t e = cudaFree(*p);
    *p = nullptr;
    *have = 0;
    if (e != cudaSuccess) return e;
  }
  size_t cap = want + want / 8 + 256;
  cudaError_t e = cudaMalloc(p, cap);
  if (e != cudaSuccess) { *p = nullptr; return e; }
  *have = cap;
  return cudaSuccess;
}

// g_mu held.  Frees the retired buffers whose last user has finished.
static void sweep_retired(DeviceCache& dc) {
  for (size_t i = 0; i < dc.retired.size();) {
    RetiredWs& r = dc.retired[i];
    cudaError_t q = r.done ? cudaEventQuery(r.done) : cudaErrorNotReady;
    if (q == cudaSuccess) {
      cudaFree(r.ptr);
      cudaEventDestroy(r.done);
      dc.retired[i] = dc.retired.back();
      dc.retired.pop_back();
    } else {
      if (q != cudaErrorNotReady) cudaGetLastError();  // an event that cannot be queried: the buffer stays until nacl_release
      ++i;
    }
  }
}

// g_mu held.  The buffer of `w` leaves service: freed once w.done has completed (never, if a graph may hold it).
static void retire(DeviceCache& dc, WsEntry& w) {
  if (w.captured) {
    dc.retired.push_back(RetiredWs{w.ptr, nullptr});
    if (w.done) cudaEventDestroy(w.done);
  } else {
    dc.retired.push_back(RetiredWs{w.ptr, w.done});
  }
  w.ptr = nullptr;
  w.done = nullptr;
}

// g_mu held
static cudaError_t stream_workspace(DeviceCache& dc, cudaStream_t st, size_t want, void** out, size_t** sync_clean = nullptr) {
  sweep_retired(dc);
  const size_t cap = want + want / 8 + 256;
  for (WsEntry& w : dc.ws)
    if (w.stream == st) {
      if (sync_clean) *sync_clean = &w.sync_clean;
      w.last_use = ++dc.tick;
      if (w.bytes < want) {
        void* np = nullptr;
        cudaEvent_t ne = nullptr;
        cudaError_t e = cudaMalloc(&np, cap);
        if (e != cudaSuccess) return e;
        if ((e = cudaEventCreateWithFlags(&ne, cudaEventDisableTiming)) != cudaSuccess) { cudaFree(np); return e; }
        retire(dc, w);
        w.ptr = np;
        w.done = ne;
        w.bytes = cap;
        w.sync_clean = 0;
        w.captured = false;
      }
      *out = w.ptr;
      return cudaSuccess;
    }
  void* np = nullptr;
  cudaEvent_t ne = nullptr;
  cudaError_t e = cudaMalloc(&np, cap);
  if (e != cudaSuccess) return e;
  if ((e = cudaEventCreateWithFlags(&ne, cudaEventDisableTiming)) != cudaSuccess) { cudaFree(np); return e; }
  if (dc.ws.size() >= kMaxStreamWorkspaces) {
    // the stream that has gone unused the longest gives up its workspace (it gets a new one if it ever comes back)
    size_t lru = 0;
    for (size_t i = 1; i < dc.ws.size(); ++i)
      if (dc.ws[i].last_use < dc.ws[lru].last_use) lru = i;
    retire(dc, dc.ws[lru]);
    dc.ws[lru] = dc.ws.back();
    dc.ws.pop_back();
  }
  dc.ws.push_back(WsEntry{st, np, cap, 0, ne, ++dc.tick, false});
  if (sync_clean) *sync_clean = &dc.ws.back().sync_clean;
  *out = np;
  return cudaSuccess;
}

// Behind the last kernel of a call that worked in the library's workspace of (dev, st): marks the point after which that
// buffer is free to go.  Under stream capture nothing is recorded: the buffer is pinned instead (a graph may replay it).
static void workspace_call_done(int dev, cudaStream_t st) {
  cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
  if (cudaStreamIsCapturing(st, &cs) != cudaSuccess) { cudaGetLastError(); cs = cudaStreamCaptureStatusActive; }
  std::lock_guard<std::mutex> lk(g_mu);
  for (WsEntry& w : g_cache[dev].ws)
    if (w.stream == st) {
      if (cs != cudaStreamCaptureStatusNone) w.captured = true;
      else if (w.done && cudaEventRecord(w.done, st) != cudaSuccess) { cudaGetLastError(); w.captured = true; }
      return;
    }
}

static int fail_cuda(cudaError_t e) {
  g_last_cuda_error = (int)e;
  cudaGetLastError();  // clear the sticky-free error state
  return NACL_ERR_CUDA;
}

// ------------------------------------------------------------------ the call
// idx_in_ws: the index list goes to the workspace's idx_tmp (p.out_idx is ignored) and *idx_in_ws receives where that is
// (nacl_evict_generation without out_idx: this call alone decides which workspace it is and keeps its bookkeeping)
static int evict_core(const nacl_params_t& p, int32_t** idx_in_ws, int* internal_ws_dev, bool lse_only);

// lse_only (nacl_proxy_lse): steps a1-a2 alone -> p.out_lse; V, the budgets and the other outputs are not looked at
static int evict_impl(const nacl_params_t& p, int32_t** idx_in_ws = nullptr, bool lse_only = false) {
  int dev = -1;  // >= 0 once the call works in the library's own workspace of that device
  const int rc = evict_core(p, idx_in_ws, &dev, lse_only);
  // whatever was enqueued (also before an error) is the buffer's latest use
  if (dev >= 0) workspace_call_done(dev, static_cast<cudaStream_t>(p.stream));
  return rc;
}

static int evict_core(const nacl_params_t& p_in, int32_t** idx_in_ws, int* internal_ws_dev, bool lse_only) {
  nacl_params_t p = p_in;
  if (lse_only) {
    if (!p.K || !p.Qproxy || !p.out_lse) return NACL_ERR_NULL;
    if (p.lse_in || p.out_importance) return NACL_ERR_UNSUPPORTED;
    if (p.flags & ~(NACL_FLAG_CAUSAL | NACL_FLAG_SCORE_CUDA_CORES)) return NACL_ERR_UNSUPPORTED;
    // everything behind the statistics is switched off: V stands in as K (never read), empty budget, no outputs
    p.V = p.K;
    p.budget_proxy = p.budget_random = p.n_sink = p.n_recent = p.n_protect = 0;
    p.protect_idx = nullptr;
    p.out_K = p.out_V = nullptr;
    p.out_idx = nullptr;
    p.out_stride_batch = p.out_stride_head = p.out_stride_row = 0;
    p.flags |= NACL_FLAG_SCORE_TWO_LAUNCHES;  // no hand-over counters in this form
  }
  if (!p.K || !p.V || !p.Qproxy) return NACL_ERR_NULL;
  // an empty budget (C == 0) has empty outputs: their pointers may be NULL
  const bool empty_out = p.budget_proxy == 0 && p.budget_random == 0;
  if (!empty_out && (!p.out_K || !p.out_V || (!p.out_idx && !idx_in_ws))) return NACL_ERR_NULL;
  int rc = validate_shape(p.dtype, p.batch, p.L, p.Hq, p.Hkv, p.d, p.P);
  if (rc) return rc;
  rc = validate_budget(p.L, p.budget_proxy, p.budget_random, p.n_sink, p.n_recent, p.n_protect);
  if (rc) return rc;
  if (p.n_protect > 0 && !p.protect_idx) return NACL_ERR_NULL;
  if (p.reserved0 != 0) return NACL_ERR_UNSUPPORTED;
  const uint32_t known = NACL_FLAG_CAUSAL | NACL_FLAG_SAMPLE_SOFTMAX_OF_SCORE | NACL_FLAG_SAMPLE_UNIFORM | NACL_FLAG_SHARED_HEADS |
                         NACL_FLAG_SCORE_CUDA_CORES | NACL_FLAG_SCORE_TWO_LAUNCHES | NACL_FLAG_SELECT_GENERAL | NACL_FLAG_GATHER_SEPARATE | NACL_FLAG_SELECT_SHARE_SMS;
  if (p.flags & ~known) return NACL_ERR_UNSUPPORTED;
  if ((p.flags & NACL_FLAG_SAMPLE_SOFTMAX_OF_SCORE) && (p.flags & NACL_FLAG_SAMPLE_UNIFORM)) return NACL_ERR_UNSUPPORTED;

  Shape s;
  s.batch = p.batch; s.L = p.L; s.Hq = p.Hq; s.Hkv = p.Hkv; s.d = p.d; s.P = p.P;
  s.G = p.Hq / p.Hkv; s.rows = s.G * p.P; s.dtype = p.dtype; s.esize = p.dtype == NACL_DTYPE_F32 ? 4 : 2;
  const int row_bytes = s.d * s.esize;
  if (row_bytes % 16 != 0) return NACL_ERR_ALIGN;
  const int C = p.budget_proxy + p.budget_random;
  // layouts: all-zero strides = contiguous
  {
    const bool kv0 = p.kv_stride_batch == 0 && p.kv_stride_head == 0 && p.kv_stride_row == 0;
    const bool o0 = p.out_stride_batch == 0 && p.out_stride_head == 0 && p.out_stride_row == 0;
    if (!kv0 && !p.block_table && (p.kv_stride_batch <= 0 || p.kv_stride_head <= 0 || p.kv_stride_row < p.d)) return NACL_ERR_SHAPE;
    if (!o0 && (p.out_stride_batch <= 0 || p.out_stride_head <= 0 || p.out_stride_row < p.d)) return NACL_ERR_SHAPE;
    s.kv_sr = kv0 ? p.d : p.kv_stride_row;
    s.kv_sh = kv0 ? (long long)p.L * p.d : p.kv_stride_head;
    s.kv_sb = kv0 ? (long long)p.Hkv * p.L * p.d : p.kv_stride_batch;
    s.o_sr = o0 ? p.d : p.out_stride_row;
    s.o_sh = o0 ? (long long)C * p.d : p.out_stride_head;
    s.o_sb = o0 ? (long long)p.Hkv * C * p.d : p.out_stride_batch;
    const long long epv = 16 / s.esize;
    if (s.kv_sr % epv || s.kv_sh % epv || s.kv_sb % epv || s.o_sr % epv || s.o_sh % epv || s.o_sb % epv) return NACL_ERR_ALIGN;
  }
  if (p.block_table) {
    if (p.reserved1 != 0) return NACL_ERR_UNSUPPORTED;
    const int ps = p.page_size;
    if (!(ps == 8 || ps == 16 || ps == 32 || ps == 64 || ps == 128) || p.n_pages < 1) return NACL_ERR_SHAPE;
    if ((long long)p.table_stride * ps < p.L) return NACL_ERR_SHAPE;
    if (reinterpret_cast<uintptr_t>(p.block_table) & 3u) return NACL_ERR_ALIGN;
    const bool pg0 = p.kv_stride_page == 0 && p.kv_stride_head == 0 && p.kv_stride_row == 0;
    if (!pg0 && (p.kv_stride_page <= 0 || p.kv_stride_head <= 0 || p.kv_stride_row < p.d)) return NACL_ERR_SHAPE;
    s.table = p.block_table; s.ps = ps; s.tstride = p.table_stride; s.n_pages = p.n_pages;
    s.kv_sr = pg0 ? p.d : p.kv_stride_row;
    s.kv_sh = pg0 ? (long long)ps * p.d : p.kv_stride_head;
    s.kv_sp = pg0 ? (long long)p.Hkv * ps * p.d : p.kv_stride_page;
    s.kv_sb = 0;
    const long long epv = 16 / s.esize;
    if (s.kv_sr % epv || s.kv_sh % epv || s.kv_sp % epv) return NACL_ERR_ALIGN;
    // only the tensor-core scoring kernel walks a block table
    if ((p.flags & NACL_FLAG_SCORE_CUDA_CORES) || !score_tc_supported(s)) return NACL_ERR_UNSUPPORTED;
  } else if (p.page_size != 0 || p.table_stride != 0 || p.n_pages != 0 || p.kv_stride_page != 0 || p.reserved1 != 0) {
    return NACL_ERR_UNSUPPORTED;
  }
  if (!aligned16(p.K) || !aligned16(p.V) || !aligned16(p.Qproxy) || !aligned16(p.out_K) || !aligned16(p.out_V) ||
      (!idx_in_ws && (reinterpret_cast<uintptr_t>(p.out_idx) & 3u)))
    return NACL_ERR_ALIGN;

  if (p.batch_offset < 0 || p.head_offset < 0) return NACL_ERR_SHAPE;
  // in-place compaction: the compacted cache takes the first C rows of every head of the SAME buffers
  bool inplace = false;
  if (!empty_out && (p.out_K == p.K || p.out_V == p.V)) {
    if (p.out_K != p.K || p.out_V != p.V || p.block_table || (p.flags & NACL_FLAG_SHARED_HEADS) || s.o_sr != s.kv_sr ||
        s.o_sh != s.kv_sh || s.o_sb != s.kv_sb || s.kv_sr != s.d)
      return NACL_ERR_UNSUPPORTED;
    inplace = true;
  }
  const size_t need = nacl_workspace_bytes(p.batch, p.L, p.Hq, p.Hkv, p.d, p.P);
  cudaStream_t st = static_cast<cudaStream_t>(p.stream);
  cudaError_t e;
  void* wsp = p.workspace;
  const bool tc = !(p.flags & NACL_FLAG_SCORE_CUDA_CORES) && score_tc_supported(s);
  const bool two_launches = (p.flags & NACL_FLAG_SCORE_TWO_LAUNCHES) != 0;
  // the fused scoring launch hands the softmax partials from CTA to CTA through counters that must be zero at launch;
  // the kernel leaves them zero again.  A caller's workspace is zeroed every time, the library's own only when the
  // counters reach into bytes that another shape may have used for something else.
  const size_t sync_bytes = (tc && !two_launches && !p.lse_in) ? sync_ints((size_t)p.batch * p.Hkv) * sizeof(int) : 0;
  bool zero_sync = sync_bytes > 0;
  if (wsp) {
    if (p.workspace_bytes < need || (reinterpret_cast<uintptr_t>(wsp) & 255u)) return NACL_ERR_WORKSPACE;
  } else {
    int dev = 0;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return fail_cuda(e);
    if (dev < 0 || dev >= 64) return NACL_ERR_UNSUPPORTED;
    std::lock_guard<std::mutex> lk(g_mu);
    size_t* clean = nullptr;
    e = stream_workspace(g_cache[dev], st, need, &wsp, &clean);
    if (e != cudaSuccess) return fail_cuda(e);
    *internal_ws_dev = dev;
    // the counters' bytes are reserved for them in every carve-up; what lies behind them is written by this call's other buffers
    const size_t reserved = sync_ints((size_t)p.batch * p.Hkv) * sizeof(int);
    if (sync_bytes > 0) {
      if (*clean >= reserved) zero_sync = false;
      *clean = reserved;
    } else if (*clean > reserved) {
      *clean = reserved;
    }
  }
  const Workspace ws = carve_workspace(wsp, p.batch, p.L, p.Hq, p.Hkv, p.P);
  const SplitPlan sp = make_split_plan(p.batch, p.L, p.Hkv);
  int32_t* const out_idx = idx_in_ws ? ws.idx_tmp : p.out_idx;
  if (idx_in_ws) *idx_in_ws = ws.idx_tmp;
  if (zero_sync && (e = cudaMemsetAsync(ws.sync, 0, sync_bytes, st)) != cudaSuccess) return fail_cuda(e);

  if (p.lse_in && (reinterpret_cast<uintptr_t>(p.lse_in) & 3u)) return NACL_ERR_ALIGN;
  if (p.out_lse && (reinterpret_cast<uintptr_t>(p.out_lse) & 3u)) return NACL_ERR_ALIGN;
  const bool causal = (p.flags & NACL_FLAG_CAUSAL) != 0;
  if (lse_only) {
    if (tc) e = launch_score_tc(s, p.K, p.Qproxy, sp, ws, nullptr, causal, true, nullptr, p.out_lse, st, true);
    else e = launch_score_generic(s, p.K, p.Qproxy, sp, ws, nullptr, causal, nullptr, p.out_lse, st, true);
    return e == cudaSuccess ? NACL_OK : fail_cuda(e);
  }
  if (tc) e = launch_score_tc(s, p.K, p.Qproxy, sp, ws, p.lse_in, causal, two_launches, p.out_importance, p.out_lse, st);
  else e = launch_score_generic(s, p.K, p.Qproxy, sp, ws, p.lse_in, causal, p.out_importance, p.out_lse, st);
  if (e != cudaSuccess) return fail_cuda(e);

  bool gathered = false;
  if (p.flags & NACL_FLAG_SHARED_HEADS) {
    // one selection per batch element on the head-summed importance (a [batch, 1, L] problem drawn with the stream of the
    // call's first head), then the same index row for every head and the stand-alone gather
    if ((e = launch_head_sum(ws.imp, ws.imp_sh, p.batch, p.Hkv, p.L, st)) != cudaSuccess) return fail_cuda(e);
    if ((e = launch_protect(ws.imp_sh, p.batch, p.L, p.protect_idx, p.n_protect, st)) != cudaSuccess) return fail_cuda(e);
    e = launch_select(ws.imp_sh, ws.key, p.batch, 1, p.L, p.budget_proxy, p.budget_random, p.n_sink, p.n_recent, p.seed, p.layer,
                      p.flags, ws.idx_sh, nullptr, nullptr, nullptr, nullptr, row_bytes, &gathered, p.batch_offset, p.head_offset, &s,
                      (float)p.Hkv * (float)s.rows / (float)p.L, false, st);
    if (e == cudaSuccess) e = launch_replicate_idx(ws.idx_sh, out_idx, p.batch, p.Hkv, C, st);
  } else {
    if ((e = launch_protect(ws.imp, p.batch * p.Hkv, p.L, p.protect_idx, p.n_protect, st)) != cudaSuccess) return fail_cuda(e);
    e = launch_select(ws.imp, ws.key, p.batch, p.Hkv, p.L, p.budget_proxy, p.budget_random, p.n_sink, p.n_recent, p.seed, p.layer,
                      p.flags, out_idx, p.K, p.V, p.out_K, p.out_V, row_bytes, &gathered, p.batch_offset, p.head_offset, &s,
                      (float)s.rows / (float)p.L, inplace, st);
  }
  if (e == cudaErrorNotSupported && inplace) { cudaGetLastError(); return NACL_ERR_UNSUPPORTED; }  // rows too long for the fused gather
  if (e != cudaSuccess) return fail_cuda(e);
  if (!gathered) {
    StageScope sc(ST_GATHER, st);
    e = launch_gather(p.K, p.V, out_idx, s, C, row_bytes, p.out_K, p.out_V, st);
  }
  if (e != cudaSuccess) return fail_cuda(e);
  return NACL_OK;
}

static nacl_params_t make_params(int dtype, const void* K, const void* V, const void* Q, int batch, int L, int Hq, int Hkv,
                                 int d, int P, int bp, int br, int n_sink, int n_recent, uint64_t seed, int layer,
                                 void* oK, void* oV, int32_t* oidx, void* stream) {
  nacl_params_t p{};
  p.struct_size = sizeof(nacl_params_t);
  p.dtype = dtype;
  p.K = K; p.V = V; p.Qproxy = Q;
  p.batch = batch; p.L = L; p.Hq = Hq; p.Hkv = Hkv; p.d = d; p.P = P;
  p.budget_proxy = bp; p.budget_random = br; p.n_sink = n_sink; p.n_recent = n_recent;
  p.seed = seed; p.layer = layer; p.flags = 0;
  p.out_K = oK; p.out_V = oV; p.out_idx = oidx;
  p.stream = stream;
  return p;
}

// ------------------------------------------------------------------ nacl_evict_static: the call that allocates nothing
// Scratch for callers that cannot allocate device memory (see include/nacl_evict.h).  It lives in the library's own
// device image: every GPU that loads libnacl_evict.so holds these NACL_STATIC_SCRATCH_BYTES from module load to exit.
// NOTE for maintainers: in HOST code the name g_static_scratch is only a handle for the runtime, not a device address
// (a kernel handed `g_static_scratch` from host code would fault or scribble over unrelated memory).  Kernels must be
// given the pointer that cudaGetSymbolAddress returns while the device in question is current.
static __device__ __align__(256) unsigned char g_static_scratch[NACL_STATIC_SCRATCH_BYTES];
static void* g_static_scratch_addr[64] = {};  // per device, filled by the first nacl_evict_static call there

// The array's address on the CURRENT device; looked up once per device (no allocation: the array already exists).
static int static_scratch_here(void** out) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail_cuda(e);
  if (dev < 0 || dev >= 64) return NACL_ERR_UNSUPPORTED;
  std::lock_guard<std::mutex> lk(g_mu);
  if (!g_static_scratch_addr[dev]) {
    void* addr = nullptr;
    if ((e = cudaGetSymbolAddress(&addr, g_static_scratch)) != cudaSuccess) return fail_cuda(e);
    if (!addr || (reinterpret_cast<uintptr_t>(addr) & 255u)) return NACL_ERR_WORKSPACE;
    g_static_scratch_addr[dev] = addr;
  }
  *out = g_static_scratch_addr[dev];
  return NACL_OK;
}

}  // namespace nacl

using namespace nacl;

#pragma GCC visibility push(default)
extern "C" {

int nacl_evict(const void* K, const void* V, const void* Qproxy, int batch, int L, int Hq, int Hkv, int d, int P,
               int budget_proxy, int budget_random, int n_sink, int n_recent, uint64_t seed, int layer, void* out_K,
               void* out_V, int32_t* out_idx, void* stream) {
  return evict_impl(make_params(NACL_DTYPE_BF16, K, V, Qproxy, batch, L, Hq, Hkv, d, P, budget_proxy, budget_random, n_sink,
                                n_recent, seed, layer, out_K, out_V, out_idx, stream));
}

int nacl_evict_f32(const void* K, const void* V, const void* Qproxy, int batch, int L, int Hq, int Hkv, int d, int P,
                   int budget_proxy, int budget_random, int n_sink, int n_recent, uint64_t seed, int layer, void* out_K,
                   void* out_V, int32_t* out_idx, void* stream) {
  return evict_impl(make_params(NACL_DTYPE_F32, K, V, Qproxy, batch, L, Hq, Hkv, d, P, budget_proxy, budget_random, n_sink,
                                n_recent, seed, layer, out_K, out_V, out_idx, stream));
}

int nacl_evict_ex(const nacl_params_t* p) {
  if (!p) return NACL_ERR_NULL;
  if (p->struct_size != sizeof(nacl_params_t)) return NACL_ERR_UNSUPPORTED;
  return evict_impl(*p);
}

int nacl_proxy_lse(const nacl_params_t* p) {
  if (!p) return NACL_ERR_NULL;
  if (p->struct_size != sizeof(nacl_params_t)) return NACL_ERR_UNSUPPORTED;
  return evict_impl(*p, nullptr, true);
}

int nacl_evict_static(const nacl_params_t* p) {
  if (!p) return NACL_ERR_NULL;
  if (p->struct_size != sizeof(nacl_params_t)) return NACL_ERR_UNSUPPORTED;
  if (p->workspace != nullptr || p->workspace_bytes != 0) return NACL_ERR_WORKSPACE;  // the scratch is the library's here
  // the shape decides the scratch size; an invalid shape gets its own code before any size is compared
  int rc = validate_shape(p->dtype, p->batch, p->L, p->Hq, p->Hkv, p->d, p->P);
  if (rc) return rc;
  const size_t need = nacl_workspace_bytes(p->batch, p->L, p->Hq, p->Hkv, p->d, p->P);
  if (need == 0 || need > (size_t)NACL_STATIC_SCRATCH_BYTES) return NACL_ERR_STATIC_LIMIT;
  void* scratch = nullptr;
  if ((rc = static_scratch_here(&scratch)) != NACL_OK) return rc;
  nacl_params_t q = *p;
  q.workspace = scratch;
  q.workspace_bytes = NACL_STATIC_SCRATCH_BYTES;
  // from here on this is the caller-workspace path of nacl_evict_ex: it clears the hand-over counters that must start at
  // zero on every call (cudaMemsetAsync on the stream) and overwrites everything else before reading it, so whatever an
  // earlier call of any shape left in the array does no harm
  return evict_impl(q);
}

int nacl_evict_batch(const nacl_params_t* p, int n) {
  if (n < 0 || (n > 0 && !p)) return NACL_ERR_NULL;
  if (n == 0) return NACL_OK;
  for (int i = 0; i < n; ++i) {
    if (p[i].struct_size != sizeof(nacl_params_t)) return NACL_ERR_UNSUPPORTED;
    if (p[i].stream != p[0].stream) return NACL_ERR_UNSUPPORTED;
  }
  if (n == 1) return evict_impl(p[0]);
  static std::mutex batch_mu;  // the fork / join events and the two streams are shared per device: one enqueue at a time
  std::lock_guard<std::mutex> batch_lk(batch_mu);
  cudaError_t e;
  int dev = 0;
  if ((e = cudaGetDevice(&dev)) != cudaSuccess) return fail_cuda(e);
  if (dev < 0 || dev >= 64) return NACL_ERR_UNSUPPORTED;
  cudaStream_t user = static_cast<cudaStream_t>(p[0].stream), bs[2];
  cudaEvent_t fork, join[2];
  {
    std::lock_guard<std::mutex> lk(g_mu);
    DeviceCache& dc = g_cache[dev];
    for (int sl = 0; sl < 2; ++sl) {
      if (!dc.bstream[sl] && (e = cudaStreamCreateWithFlags(&dc.bstream[sl], cudaStreamNonBlocking)) != cudaSuccess) return fail_cuda(e);
      if (!dc.bjoin[sl] && (e = cudaEventCreateWithFlags(&dc.bjoin[sl], cudaEventDisableTiming)) != cudaSuccess) return fail_cuda(e);
      bs[sl] = dc.bstream[sl];
      join[sl] = dc.bjoin[sl];
    }
    if (!dc.bfork && (e = cudaEventCreateWithFlags(&dc.bfork, cudaEventDisableTiming)) != cudaSuccess) return fail_cuda(e);
    fork = dc.bfork;
  }
  // fork: both internal streams start behind everything enqueued on the caller's stream so far
  if ((e = cudaEventRecord(fork, user)) != cudaSuccess || (e = cudaStreamWaitEvent(bs[0], fork, 0)) != cudaSuccess ||
      (e = cudaStreamWaitEvent(bs[1], fork, 0)) != cudaSuccess)
    return fail_cuda(e);
  int rc = NACL_OK;
  for (int i = 0; i < n && rc == NACL_OK; ++i) {
    nacl_params_t q = p[i];
    q.stream = bs[i & 1];
    // two plain launches for the scoring sweeps: a cooperative launch waits for ALL SMs, plain launches fill the SMs the
    // other stream's selection / gather leaves idle
    q.flags |= NACL_FLAG_SCORE_TWO_LAUNCHES | NACL_FLAG_SELECT_SHARE_SMS;
    rc = evict_impl(q);
  }
  // join (also after an error: the caller's stream must not run ahead of what was enqueued)
  for (int sl = 0; sl < 2; ++sl)
    if ((e = cudaEventRecord(join[sl], bs[sl])) != cudaSuccess || (e = cudaStreamWaitEvent(user, join[sl], 0)) != cudaSuccess)
      return rc != NACL_OK ? rc : fail_cuda(e);
  return rc;
}

int nacl_evict_generation(const nacl_gen_params_t* g) {
  if (!g) return NACL_ERR_NULL;
  if (g->struct_size != sizeof(nacl_gen_params_t)) return NACL_ERR_UNSUPPORTED;
  if (!g->K_cache || !g->V_cache || !g->q || !g->K_out || !g->V_out) return NACL_ERR_NULL;
  if ((g->pos_in == nullptr) != (g->pos_out == nullptr)) return NACL_ERR_NULL;
  if (g->reserved0 != 0 || (g->flags & NACL_FLAG_CAUSAL)) return NACL_ERR_UNSUPPORTED;  // one query row: nothing to mask
  if (g->len < 1 || g->cap_in < g->len || g->step < 0) return NACL_ERR_SHAPE;
  const long C = (long)g->budget_proxy + g->budget_random;
  if (g->budget_proxy < 0 || g->budget_random < 0 || g->cap_out < C) return NACL_ERR_BUDGET;
  int rc = validate_shape(g->dtype, g->batch, g->len, g->Hq, g->Hkv, g->d, 1);
  if (rc) return rc;
  nacl_params_t p{};
  p.struct_size = sizeof(nacl_params_t);
  p.dtype = g->dtype;
  p.K = g->K_cache; p.V = g->V_cache; p.Qproxy = g->q;
  p.batch = g->batch; p.L = g->len; p.Hq = g->Hq; p.Hkv = g->Hkv; p.d = g->d; p.P = 1;
  p.budget_proxy = g->budget_proxy; p.budget_random = g->budget_random; p.n_sink = g->n_sink; p.n_recent = g->n_recent;
  p.seed = g->seed + (uint64_t)g->step * 0x9E3779B97F4A7C15ull;  // an independent stream per decoding step (R16)
  p.layer = g->layer; p.flags = g->flags;
  p.out_K = g->K_out; p.out_V = g->V_out;
  p.out_importance = g->out_importance;
  p.workspace = g->workspace; p.workspace_bytes = g->workspace_bytes; p.stream = g->stream;
  p.batch_offset = g->batch_offset; p.head_offset = g->head_offset;
  p.kv_stride_row = g->d; p.kv_stride_head = (int64_t)g->cap_in * g->d; p.kv_stride_batch = (int64_t)g->Hkv * g->cap_in * g->d;
  p.out_stride_row = g->d; p.out_stride_head = (int64_t)g->cap_out * g->d; p.out_stride_batch = (int64_t)g->Hkv * g->cap_out * g->d;
  // without out_idx the kept slots are still needed for the position map: evict_impl then writes them to its workspace
  // (the caller's or the library's own, chosen and accounted for there as for any other call) and says where
  int32_t* idx = g->out_idx;
  p.out_idx = idx;
  if (!idx && C > 0) rc = evict_impl(p, &idx);
  else rc = evict_impl(p);
  if (rc != NACL_OK || !g->pos_in || C == 0) return rc;
  cudaError_t e = launch_compose_positions(g->pos_in, g->cap_in, idx, g->batch * g->Hkv, (int)C, g->pos_out, g->cap_out,
                                           static_cast<cudaStream_t>(g->stream));
  if (!g->out_idx && !g->workspace) {
    // this kernel read the kept slots out of the library's workspace: it is that buffer's latest use now
    int dev = -1;
    if (cudaGetDevice(&dev) == cudaSuccess && dev >= 0 && dev < 64) workspace_call_done(dev, static_cast<cudaStream_t>(g->stream));
    else cudaGetLastError();
  }
  return e == cudaSuccess ? NACL_OK : fail_cuda(e);
}

int nacl_evict_varlen(const nacl_params_t* p, const int32_t* seq_len, const int32_t* budget_proxy, const int32_t* budget_random,
                      int C_max) {
  if (!p || !seq_len || !budget_proxy || !budget_random) return NACL_ERR_NULL;
  if (p->struct_size != sizeof(nacl_params_t)) return NACL_ERR_UNSUPPORTED;
  if (p->lse_in || p->out_importance || p->out_lse || p->protect_idx || p->n_protect != 0 || p->block_table) return NACL_ERR_UNSUPPORTED;
  if (p->batch < 1 || p->L < 1 || p->Hkv < 1 || p->Hq < 1 || p->d < 1 || p->P < 1 || C_max < 0) return NACL_ERR_SHAPE;
  const size_t esz = p->dtype == NACL_DTYPE_F32 ? 4 : 2;
  // element strides of the padded tensors (all-zero = contiguous [batch, Hkv, L, d] / [batch, Hkv, C_max, d])
  const bool kv0 = p->kv_stride_batch == 0 && p->kv_stride_head == 0 && p->kv_stride_row == 0;
  const bool o0 = p->out_stride_batch == 0 && p->out_stride_head == 0 && p->out_stride_row == 0;
  const int64_t kv_sr = kv0 ? p->d : p->kv_stride_row, kv_sh = kv0 ? (int64_t)p->L * p->d : p->kv_stride_head;
  const int64_t kv_sb = kv0 ? (int64_t)p->Hkv * p->L * p->d : p->kv_stride_batch;
  const int64_t o_sr = o0 ? p->d : p->out_stride_row, o_sh = o0 ? (int64_t)C_max * p->d : p->out_stride_head;
  const int64_t o_sb = o0 ? (int64_t)p->Hkv * C_max * p->d : p->out_stride_batch;
  // every element is checked before anything is enqueued: no output is written on a validation error
  for (int b = 0; b < p->batch; ++b) {
    if (seq_len[b] < 1 || seq_len[b] > p->L) return NACL_ERR_SHAPE;
    if (budget_proxy[b] < 0 || budget_random[b] < 0 || (long)budget_proxy[b] + budget_random[b] > C_max) return NACL_ERR_BUDGET;
    int rc = validate_shape(p->dtype, 1, seq_len[b], p->Hq, p->Hkv, p->d, p->P);  // P > seq_len[b] among others
    if (rc) return rc;
    if ((rc = validate_budget(seq_len[b], budget_proxy[b], budget_random[b], p->n_sink, p->n_recent)) != NACL_OK) return rc;
  }
  for (int b = 0; b < p->batch; ++b) {
    if (budget_proxy[b] + budget_random[b] == 0) continue;  // keeps nothing: no output rows, nothing to compute
    nacl_params_t q = *p;
    q.batch = 1;
    q.L = seq_len[b];
    q.budget_proxy = budget_proxy[b];
    q.budget_random = budget_random[b];
    q.batch_offset = p->batch_offset + b;
    q.K = static_cast<const char*>(p->K) + (size_t)b * kv_sb * esz;
    q.V = static_cast<const char*>(p->V) + (size_t)b * kv_sb * esz;
    q.Qproxy = static_cast<const char*>(p->Qproxy) + (size_t)b * p->Hq * p->P * p->d * esz;
    q.out_K = p->out_K ? static_cast<char*>(p->out_K) + (size_t)b * o_sb * esz : nullptr;
    q.out_V = p->out_V ? static_cast<char*>(p->out_V) + (size_t)b * o_sb * esz : nullptr;
    q.out_idx = p->out_idx ? p->out_idx + (size_t)b * p->Hkv * C_max : nullptr;
    q.kv_stride_row = kv_sr; q.kv_stride_head = kv_sh; q.kv_stride_batch = kv_sb;
    q.out_stride_row = o_sr; q.out_stride_head = o_sh; q.out_stride_batch = o_sb;
    const int rc = evict_impl(q);
    if (rc != NACL_OK) return rc;
  }
  return NACL_OK;
}

// n problems of one shape out of HOST memory, pipelined over two staging slots with a stream each: the host-to-device
// copies of problem i+1 run under the kernels and the device-to-host copies of problem i (separate copy engines).
static int evict_host_impl(int n, const void* const* K, const void* const* V, const void* const* Qproxy, int dtype, int batch, int L,
                           int Hq, int Hkv, int d, int P, int budget_proxy, int budget_random, int n_sink, int n_recent,
                           const uint64_t* seed, const int32_t* layer, void* const* out_K, void* const* out_V,
                           int32_t* const* out_idx, int device) {
  if (n < 0 || (n > 0 && (!K || !V || !Qproxy || !seed || !layer))) return NACL_ERR_NULL;
  const bool empty_out = budget_proxy == 0 && budget_random == 0;  // empty outputs: their pointers may be NULL
  if (n > 0 && !empty_out && (!out_K || !out_V || !out_idx)) return NACL_ERR_NULL;
  for (int i = 0; i < n; ++i) {
    if (!K[i] || !V[i] || !Qproxy[i]) return NACL_ERR_NULL;
    if (!empty_out && (!out_K[i] || !out_V[i] || !out_idx[i])) return NACL_ERR_NULL;
  }
  int rc = validate_shape(dtype, batch, L, Hq, Hkv, d, P);
  if (rc) return rc;
  rc = validate_budget(L, budget_proxy, budget_random, n_sink, n_recent);
  if (rc) return rc;
  if (n == 0) return NACL_OK;
  std::lock_guard<std::mutex> host_lk(g_host_mu);
  cudaError_t e;
  int prev = -1;
  if ((e = cudaGetDevice(&prev)) != cudaSuccess) return fail_cuda(e);
  if (device < 0) device = prev;
  if (device >= 64) return NACL_ERR_UNSUPPORTED;
  if (device != prev && (e = cudaSetDevice(device)) != cudaSuccess) return fail_cuda(e);

  const size_t esz = dtype == NACL_DTYPE_F32 ? 4 : 2;
  const int C = budget_proxy + budget_random;
  const size_t kv_bytes = (size_t)batch * Hkv * L * d * esz;
  const size_t q_bytes = (size_t)batch * Hq * P * d * esz;
  const size_t okv_bytes = (size_t)batch * Hkv * C * d * esz;
  const size_t idx_bytes = (size_t)batch * Hkv * C * sizeof(int32_t);
  const size_t want[6] = {kv_bytes, kv_bytes, q_bytes, okv_bytes, okv_bytes, idx_bytes};
  const int n_slots = n > 1 ? 2 : 1;

  std::unique_lock<std::mutex> lk(g_mu);
  DeviceCache& dc = g_cache[device];
  rc = NACL_OK;
  for (int sl = 0; sl < n_slots && rc == NACL_OK; ++sl) {
    for (int i = 0; i < 6 && rc == NACL_OK; ++i)
      if ((e = grow(&dc.stage[sl][i], &dc.stage_bytes[sl][i], want[i] ? want[i] : 16)) != cudaSuccess) rc = fail_cuda(e);
    if (rc == NACL_OK && !dc.stream[sl] && (e = cudaStreamCreateWithFlags(&dc.stream[sl], cudaStreamNonBlocking)) != cudaSuccess)
      rc = fail_cuda(e);
  }
  void* stg[2][6];
  cudaStream_t sts[2] = {dc.stream[0], dc.stream[1]};
  for (int sl = 0; sl < 2; ++sl)
    for (int i = 0; i < 6; ++i) stg[sl][i] = dc.stage[sl][i];
  lk.unlock();

  for (int i = 0; i < n && rc == NACL_OK; ++i) {
    const int sl = i % n_slots;
    cudaStream_t st = sts[sl];
    void* sK = stg[sl][0]; void* sV = stg[sl][1]; void* sQ = stg[sl][2];
    void* soK = stg[sl][3]; void* soV = stg[sl][4]; void* sidx = stg[sl][5];
    // one cudaMemcpyAsync per tensor; pinned host memory makes them truly asynchronous.  A slot's buffers are reused in
    // stream order: problem i waits for problem i - 2 on the same stream
    if ((e = cudaMemcpyAsync(sQ, Qproxy[i], q_bytes, cudaMemcpyHostToDevice, st)) != cudaSuccess ||
        (e = cudaMemcpyAsync(sK, K[i], kv_bytes, cudaMemcpyHostToDevice, st)) != cudaSuccess ||
        (e = cudaMemcpyAsync(sV, V[i], kv_bytes, cudaMemcpyHostToDevice, st)) != cudaSuccess) {
      rc = fail_cuda(e);
      break;
    }
    nacl_params_t p = make_params(dtype, sK, sV, sQ, batch, L, Hq, Hkv, d, P, budget_proxy, budget_random, n_sink, n_recent,
                                  seed[i], layer[i], soK, soV, static_cast<int32_t*>(sidx), st);
    rc = evict_impl(p);
    if (rc == NACL_OK && C > 0) {
      if ((e = cudaMemcpyAsync(out_idx[i], sidx, idx_bytes, cudaMemcpyDeviceToHost, st)) != cudaSuccess ||
          (e = cudaMemcpyAsync(out_K[i], soK, okv_bytes, cudaMemcpyDeviceToHost, st)) != cudaSuccess ||
          (e = cudaMemcpyAsync(out_V[i], soV, okv_bytes, cudaMemcpyDeviceToHost, st)) != cudaSuccess)
        rc = fail_cuda(e);
    }
  }
  for (int sl = 0; sl < n_slots; ++sl)
    if ((e = cudaStreamSynchronize(sts[sl])) != cudaSuccess && rc == NACL_OK) rc = fail_cuda(e);
  if (device != prev) cudaSetDevice(prev);
  return rc;
}

int nacl_evict_host(const void* K, const void* V, const void* Qproxy, int dtype, int batch, int L, int Hq, int Hkv, int d,
                    int P, int budget_proxy, int budget_random, int n_sink, int n_recent, uint64_t seed, int layer,
                    void* out_K, void* out_V, int32_t* out_idx, int device) {
  if (!K || !V || !Qproxy) return NACL_ERR_NULL;
  const int32_t layer32 = layer;
  return evict_host_impl(1, &K, &V, &Qproxy, dtype, batch, L, Hq, Hkv, d, P, budget_proxy, budget_random, n_sink, n_recent, &seed,
                         &layer32, &out_K, &out_V, &out_idx, device);
}

int nacl_evict_host_batch(int n, const void* const* K, const void* const* V, const void* const* Qproxy, int dtype, int batch, int L,
                          int Hq, int Hkv, int d, int P, int budget_proxy, int budget_random, int n_sink, int n_recent,
                          const uint64_t* seed, const int32_t* layer, void* const* out_K, void* const* out_V,
                          int32_t* const* out_idx, int device) {
  return evict_host_impl(n, K, V, Qproxy, dtype, batch, L, Hq, Hkv, d, P, budget_proxy, budget_random, n_sink, n_recent, seed, layer,
                         out_K, out_V, out_idx, device);
}

int nacl_gumbel_keys(const float* importance, float* out_keys, int batch, int Hkv, int L, uint64_t seed, int layer,
                     uint32_t flags, void* stream) {
  if (!importance || !out_keys) return NACL_ERR_NULL;
  if (batch < 1 || Hkv < 1 || L < 1 || L > (1 << 24) || (long)batch * Hkv > 65535) return NACL_ERR_SHAPE;
  if ((reinterpret_cast<uintptr_t>(importance) | reinterpret_cast<uintptr_t>(out_keys)) & 3u) return NACL_ERR_ALIGN;
  const uint32_t known = NACL_FLAG_SAMPLE_SOFTMAX_OF_SCORE | NACL_FLAG_SAMPLE_UNIFORM;
  if ((flags & ~known) || flags == known) return NACL_ERR_UNSUPPORTED;
  cudaError_t e = launch_keys(importance, reinterpret_cast<uint32_t*>(out_keys), batch, Hkv, L, seed, layer, flags, false, 0, 0,
                              static_cast<cudaStream_t>(stream));
  return e == cudaSuccess ? NACL_OK : fail_cuda(e);
}

size_t nacl_workspace_bytes(int batch, int L, int Hq, int Hkv, int d, int P) {
  if (validate_shape(NACL_DTYPE_BF16, batch, L, Hq, Hkv, d, P) != NACL_OK) return 0;
  return carve_workspace(nullptr, batch, L, Hq, Hkv, P).bytes;
}

int nacl_profile_enable(int on) {
  std::lock_guard<std::mutex> lk(g_prof_mu);
  g_prof_on = on != 0;
  return NACL_OK;
}

int nacl_profile_read(double* ms, int64_t* launches, int reset) {
  std::lock_guard<std::mutex> lk(g_prof_mu);
  int rc = NACL_OK;
  for (const ProfRecord& r : g_prof_pending) {
    float t = 0.f;
    cudaError_t e = cudaEventSynchronize(r.b);
    if (e == cudaSuccess) e = cudaEventElapsedTime(&t, r.a, r.b);
    if (e != cudaSuccess) { rc = fail_cuda(e); }
    else { g_prof_ms[r.stage] += (double)t; g_prof_n[r.stage] += 1; }
    g_prof_free.push_back(r.a);
    g_prof_free.push_back(r.b);
  }
  g_prof_pending.clear();
  for (int s = 0; s < ST_COUNT; ++s) {
    if (ms) ms[s] = g_prof_ms[s];
    if (launches) launches[s] = g_prof_n[s];
    if (reset) { g_prof_ms[s] = 0; g_prof_n[s] = 0; }
  }
  return rc;
}

const char* nacl_stage_name(int stage) {
  switch (stage) {
    case ST_STATS: return "score_stats";
    case ST_COMBINE: return "score_combine";
    case ST_COLSUM: return "score_colsum";
    case ST_KEYS: return "gumbel_keys";
    case ST_SELECT: return "select";
    case ST_GATHER: return "gather";
    case ST_FUSED: return "score_fused";
    default: return "?";
  }
}

void nacl_release(void) {
  std::lock_guard<std::mutex> lk(g_mu);
  int prev = -1;
  if (cudaGetDevice(&prev) != cudaSuccess) { cudaGetLastError(); return; }
  for (int dev = 0; dev < 64; ++dev) {
    DeviceCache& dc = g_cache[dev];
    bool any = !dc.ws.empty() || !dc.retired.empty() || dc.stream[0] || dc.stream[1] || dc.bstream[0] || dc.bfork;
    for (int i = 0; i < 12; ++i) any = any || dc.stage[i / 6][i % 6];
    if (!any) continue;
    if (cudaSetDevice(dev) != cudaSuccess) { cudaGetLastError(); continue; }
    cudaDeviceSynchronize();  // retired workspaces may still be in use by enqueued calls
    for (WsEntry& w : dc.ws) { cudaFree(w.ptr); if (w.done) cudaEventDestroy(w.done); }
    for (RetiredWs& r : dc.retired) { cudaFree(r.ptr); if (r.done) cudaEventDestroy(r.done); }
    for (int i = 0; i < 12; ++i) if (dc.stage[i / 6][i % 6]) cudaFree(dc.stage[i / 6][i % 6]);
    for (int sl = 0; sl < 2; ++sl) if (dc.stream[sl]) cudaStreamDestroy(dc.stream[sl]);
    for (int sl = 0; sl < 2; ++sl) if (dc.bstream[sl]) cudaStreamDestroy(dc.bstream[sl]);
    if (dc.bfork) cudaEventDestroy(dc.bfork);
    for (int sl = 0; sl < 2; ++sl) if (dc.bjoin[sl]) cudaEventDestroy(dc.bjoin[sl]);
    dc = DeviceCache();
  }
  cudaSetDevice(prev);
  cudaGetLastError();
}

const char* nacl_strerror(int code) {
  switch (code) {
    case NACL_OK: return "ok";
    case NACL_ERR_NULL: return "a required pointer is NULL";
    case NACL_ERR_SHAPE: return "unsupported shape (sizes, Hq % Hkv, P > L, d, L > 2^24)";
    case NACL_ERR_BUDGET: return "budget error (negative count, protected > L, budget_proxy < protected, total > L)";
    case NACL_ERR_ALIGN: return "pointer not 16-byte aligned or row size not a multiple of 16 bytes";
    case NACL_ERR_WORKSPACE: return "workspace too small or not 256-byte aligned";
    case NACL_ERR_CUDA: return "a CUDA call failed (see nacl_last_cuda_error)";
    case NACL_ERR_UNSUPPORTED: return "flag, dtype or struct version not supported by this build";
    case NACL_ERR_STATIC_LIMIT: return "problem needs more scratch than nacl_evict_static's built-in NACL_STATIC_SCRATCH_BYTES (use nacl_evict_ex with a workspace)";
    default: return "unknown error code";
  }
}

int nacl_last_cuda_error(void) { return g_last_cuda_error; }
int nacl_version(void) { return NACL_VERSION; }

}  // extern "C"
#pragma GCC visibility pop
