// nacl_internal.cuh -- declarations shared by the translation units of libnacl_evict.so.
// Product code (CUDA path).  Nothing here is shared with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <stddef.h>
#include <stdint.h>

#include "nacl_evict.h"

namespace nacl {

constexpr int kNumSMs = 148;  // B200; grid sizing and the workspace formula assume it

// ------------------------------------------------------------------ shape / plan
struct Shape {
  int batch, L, Hq, Hkv, d, P;
  int G;        // Hq / Hkv
  int rows;     // G * P proxy rows per kv head
  int dtype;    // NACL_DTYPE_*
  int esize;    // bytes per element
  // element strides of K and V (batch, kv head, key row; the d elements of a row are contiguous) and of out_K / out_V
  long long kv_sb, kv_sh, kv_sr, o_sb, o_sh, o_sr;
  // paged K/V (table != nullptr): position j of batch element b = row j % ps of page table[b * tstride + j / ps];
  // kv_sp = element stride between pages (kv_sb unused)
  const int32_t* table = nullptr;
  int ps = 0, tstride = 0, n_pages = 0;
  long long kv_sp = 0;
};

// How L is split for the split-L softmax statistics (a pure function of the shape).
struct SplitPlan {
  int chunk;     // keys per chunk (multiple of 128)
  int n_chunks;  // ceil(L / chunk)
};
SplitPlan make_split_plan(int batch, int L, int Hkv);

// Workspace carve-up (all offsets 256-byte aligned).
struct Workspace {
  float2* part;        // partial softmax statistics (m, Z): generic path [batch*Hq*P, n_chunks]; tensor-core path
                       // [148 + heads, n_slots, G*P] (score_tc.cu)
  float* lse;          // [batch*Hq*P]            natural-log LSE of every proxy row
  float* imp;          // [batch*Hkv, L]          importance F_score
  uint32_t* key;       // select scratch (select_scratch_words): global radix histograms, or [batch*Hkv, L] keys for very long rows
  int* sync;           // [sync_ints(heads)]      fused scoring launch: per-head hand-over counters (score_tc.cu); zero between calls
  float* imp_sh;       // [batch, L]              NACL_FLAG_SHARED_HEADS: importance summed over the kv heads
  int32_t* idx_sh;     // [batch, L]              NACL_FLAG_SHARED_HEADS: the shared retained set (C <= L entries per batch element)
  int32_t* idx_tmp;    // [batch*Hkv, L]          nacl_evict_generation without out_idx: the kept slots
  size_t bytes;
};
inline size_t sync_ints(size_t heads) { return 16 + 2 * heads; }
Workspace carve_workspace(void* base, int batch, int L, int Hq, int Hkv, int P);

// ------------------------------------------------------------------ per-stage device timing (nacl_profile_*)
enum Stage { ST_STATS = 0, ST_COMBINE, ST_COLSUM, ST_KEYS, ST_SELECT, ST_GATHER, ST_FUSED, ST_COUNT };
// Brackets one kernel launch with two CUDA events on `st` while profiling is enabled; free otherwise.
struct StageScope {
  StageScope(int stage, cudaStream_t st);
  ~StageScope();
  int stage_;
  cudaStream_t st_;
  cudaEvent_t a_, b_;  // null when profiling is off
};

// ------------------------------------------------------------------ kernels (launchers)
// Each launcher enqueues on `st` and returns the cudaError_t of the launch.

// generic CUDA-core scoring (any dtype / d / G*P): 3 launches
// lse_in != nullptr: the row log-sum-exps are given (natural log): the statistics sweep is skipped.
// causal: NACL_FLAG_CAUSAL (proxy row i = prompt position L-P+i sees keys j <= L-P+i)
// stats_only (nacl_proxy_lse): the statistics sweep and its combine alone -> lse_out; no column sums, ws.imp untouched
cudaError_t launch_score_generic(const Shape& s, const void* K, const void* Q, const SplitPlan& sp,
                                 const Workspace& ws, const float* lse_in, bool causal, float* imp_out, float* lse_out, cudaStream_t st,
                                 bool stats_only = false);

// tensor-core scoring (bf16, d == 128, G*P % 16 == 0, G*P <= 256): tcgen05 + TMA
bool score_tc_supported(const Shape& s);
size_t score_tc_part_elems(int heads, int rows);  // float2 elements of Workspace::part the tensor-core path needs
cudaError_t launch_score_tc(const Shape& s, const void* K, const void* Q, const SplitPlan& sp,
                            const Workspace& ws, const float* lse_in, bool causal, bool two_launches, float* imp_out,
                            float* lse_out, cudaStream_t st, bool stats_only = false);

// Gumbel-top-k keys: key[p,j] = fl32(ln w(imp) - ln(-ln u)), order-mapped to uint32 (ordermapped) or as float bits
// batch_offset / head_offset: global indices of the call's first batch element / kv head (Philox counter words)
cudaError_t launch_keys(const float* imp, uint32_t* key, int batch, int Hkv, int L, uint64_t seed, int layer, uint32_t flags,
                        bool ordermapped, int batch_offset, int head_offset, cudaStream_t st);

// protected + top-k + Gumbel-top-k (keys fused when the row fits a cluster's shared memory) + ascending
// compaction -> out_idx.  Records its own StageScopes.  `key` is scratch for the long-row fallback.
bool select_uses_cluster(int L);
size_t select_scratch_words(int batch, int Hkv, int L);  // 4-byte words of Workspace::key
// With K/V given and the cluster path taken, the kernel also moves the kept rows (step a7) and sets *gathered.
// imp_mean: the mean importance of a row (its sum is known: G*P, or Hkv*G*P for the head-summed rows), centre of the
// bucket windows of the fast selection path; <= 0: general path only.  inplace: out_K/out_V alias K/V with the same
// strides (contiguous rows): only the fused gather of the cluster kernel can do that (cudaErrorNotSupported otherwise).
cudaError_t launch_select(const float* imp, uint32_t* key, int batch, int Hkv, int L, int budget_proxy, int budget_random,
                          int n_sink, int n_recent, uint64_t seed, int layer, uint32_t flags, int32_t* out_idx,
                          const void* K, const void* V, void* out_K, void* out_V, int row_bytes, bool* gathered,
                          int batch_offset, int head_offset, const Shape* layout, float imp_mean, bool inplace, cudaStream_t st);

// NACL_FLAG_SHARED_HEADS: out[b, j] = sum over the kv heads (in head order, fp32) of imp[b, hk, j]
cudaError_t launch_head_sum(const float* imp, float* out, int batch, int Hkv, int L, cudaStream_t st);
// NACL_FLAG_SHARED_HEADS: idx[b, hk, :] = shared[b, :] for every kv head
cudaError_t launch_replicate_idx(const int32_t* shared, int32_t* idx, int batch, int Hkv, int C, cudaStream_t st);
// explicit protected positions: imp[p, protect_idx[e]] = +inf for every problem p (the selects then keep them first)
cudaError_t launch_protect(float* imp, int n_prob, int L, const int32_t* protect_idx, int n_protect, cudaStream_t st);

// K,V <- K_S,V_S
// layout: element strides of K/V and of out_K/out_V (Shape::kv_* / o_*), batch x Hkv problems
cudaError_t launch_gather(const void* K, const void* V, const int32_t* idx, const Shape& layout, int C,
                          int row_bytes, void* out_K, void* out_V, cudaStream_t st);
// pos_out[p, c] = pos_in[p, idx[p, c]] (int32 rows of length L_in / C_out per problem, row strides given): the
// position map of a cache that is evicted again (generation phase)
cudaError_t launch_compose_positions(const int32_t* pos_in, long long in_stride, const int32_t* idx, int n_prob, int C,
                                     int32_t* pos_out, long long out_stride, cudaStream_t st);

// ------------------------------------------------------------------ small device helpers
__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}
__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// merge two (max, sum-exp) softmax partials; (m = -inf, z = 0) is the identity
__device__ __forceinline__ void merge_mz(float& m, float& z, float m2, float z2) {
  float mn = fmaxf(m, m2);
  if (mn == -INFINITY) { m = mn; z = 0.f; return; }
  z = z * expf(m - mn) + z2 * expf(m2 - mn);
  m = mn;
}

}  // namespace nacl
