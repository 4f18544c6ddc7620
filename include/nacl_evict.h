/*
 * nacl_evict.h -- C ABI of libnacl_evict.so: NACL one-shot encoding-phase KV-cache
 * eviction (arXiv 2408.03675) as hand-written sm_100a CUDA kernels.
 *
 * The operation (PAPER.md = the paper's LaTeX source, cited by line; readings R1..R15
 * in DESIGN.md section 2).  For every batch element b and kv head hk of one layer:
 *   1. proxy logits     s[i,j] = Q[b,hq,i,:] . K[b,hk,j,:] / sqrt(d)  for the G = Hq/Hkv
 *                       query heads hq = hk*G+g of the group and the P proxy rows
 *                       (Alg.1);
 *   2. importance       imp[j] = sum_{g,i} Softmax_j(s[i,:])[j]   -- F_score, a full-length
 *                       softmax per proxy row, reduced column-wise;
 *   3. protected set    Pi = [0,n_sink) U [L-n_recent,L);
 *   4. Proxy-Tokens Eviction: T = the (budget_proxy - |Pi|) positions outside Pi with the
 *                       largest imp, ties to the lower index;
 *   5. Random Eviction: U = budget_random positions drawn without replacement from the
 *                       rest with probability proportional to imp, as
 *                       Gumbel-top-k: key_j = fl32(ln imp_j - ln(-ln u_j)), u_j from
 *                       Philox4x32-10(counter=(j,hk,b,layer), key=seed), largest keys win,
 *                       ties to the lower index;
 *   6. out_idx[b,hk,:] = sorted(Pi U T U U), C = budget_proxy + budget_random entries
 *                       (PAPER.md:163, 183);
 *   7. out_K[b,hk,c,:] = K[b,hk,out_idx[c],:], out_V likewise.
 *
 * Layouts (contiguous, row-major):
 *   K, V        [batch, Hkv, L, d]     Qproxy  [batch, Hq, P, d]  (queries of the last P
 *               prompt positions, in order)
 *   out_K/out_V [batch, Hkv, C, d]     out_idx [batch, Hkv, C] int32, strictly ascending
 *   out_importance (optional) [batch, Hkv, L] fp32;  out_lse (optional) [batch, Hq, P] fp32
 * Element type: bfloat16 (nacl_evict) or IEEE fp32 (nacl_evict_f32); nacl_evict_ex takes a tag.
 * budget_* / n_* are token counts; budget_proxy INCLUDES the n_sink + n_recent protected
 * tokens (R7).
 *
 * Ownership / behaviour: every pointer of nacl_evict, nacl_evict_f32 and nacl_evict_ex is a
 * DEVICE pointer owned by the caller; inputs are read-only; outputs must not alias inputs;
 * pointers must be 16-byte aligned and d*sizeof(element) a multiple of 16.  Work is enqueued
 * on `stream` (a cudaStream_t passed as void*); the call never synchronises the host and
 * results are valid once the stream reaches that point.  With a caller-supplied workspace
 * (nacl_evict_ex) the call allocates nothing and is CUDA-graph capturable; without one an
 * internal workspace per (device, stream) is created on first use (cudaMalloc: not capturable); calls on
 * one stream share it in stream order, calls on different streams never do, so concurrent host threads are safe as
 * long as they use different streams (or pass their own workspaces).  Growth of the internal workspaces: a stream's
 * buffer is replaced by a larger one (about 9/8 of the need) when a larger shape arrives, and the old buffer is freed by
 * a later call once the work that used it has finished; the 16 most recently used streams per device keep a buffer,
 * older ones give theirs up the same way (so streams that come and go do not pile up).  Buffers that were used while
 * their stream was being captured stay until nacl_release, since a graph may still refer to them.
 * Same inputs and seed give bit-identical outputs run to run (no floating-point atomics).
 * nacl_evict_host is the same operation on HOST buffers (copies inside; synchronous).
 *
 * nacl_evict_ex with lse_in (the row log-sum-exps, e.g. from the prefill attention) runs a single sweep over K.
 *
 * With budget_proxy + budget_random == 0 the outputs are empty and their pointers may be NULL.
 *
 * Errors: 0 = OK; negative = error; nothing is thrown and no output is written on a
 * validation error.  Validation is host-side and never reads device memory.
 *
 * Supported: 1 <= P <= L <= 2^24; Hq % Hkv == 0; d a multiple of 16, d <= 256; any L (ragged
 * last tile is masked).  The tensor-core path (tcgen05 + TMA) serves bf16, d == 128 and
 * G*P a multiple of 16 up to 8192 (above 256 in blocks of 256 proxy rows, the last block masked where G*P is off that
 * grid: the paper's proxy share of 3-20 % of the prompt); every other shape runs the generic
 * CUDA-core kernels of the same library.
 */
#ifndef NACL_EVICT_H
#define NACL_EVICT_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define NACL_VERSION 20200 /* major*10000 + minor*100 + patch: ABI 2.2.0 */

#define NACL_DTYPE_F32 0
#define NACL_DTYPE_BF16 1

#define NACL_OK 0
#define NACL_ERR_NULL (-1)        /* a required pointer is NULL */
#define NACL_ERR_SHAPE (-2)       /* sizes <= 0, Hq % Hkv != 0, P > L, unsupported d, L > 2^24 */
#define NACL_ERR_BUDGET (-3)      /* negative counts, n_sink+n_recent > L, budget_proxy < protected, total > L */
#define NACL_ERR_ALIGN (-4)       /* pointer not 16-byte aligned or d*elem not a multiple of 16 */
#define NACL_ERR_WORKSPACE (-5)   /* supplied workspace too small or misaligned */
#define NACL_ERR_CUDA (-6)        /* a CUDA runtime/driver call failed; see nacl_last_cuda_error() */
#define NACL_ERR_UNSUPPORTED (-7) /* a flag or dtype this build does not implement */
#define NACL_ERR_STATIC_LIMIT (-8) /* nacl_evict_static: the shape needs more than NACL_STATIC_SCRATCH_BYTES of scratch */

/* nacl_evict_ex flags */
#define NACL_FLAG_CAUSAL 1u                  /* DESIGN.md R1: proxy row i is prompt position L-P+i and sees keys j <= L-P+i */
#define NACL_FLAG_SAMPLE_SOFTMAX_OF_SCORE 2u /* sampling weight exp(imp_j) (R4) */
#define NACL_FLAG_SAMPLE_UNIFORM 4u          /* uniform sampling weights (paper's ablation) */
#define NACL_FLAG_SHARED_HEADS 8u            /* the paper's "- Head-wise" ablation: ONE retained set
                                                per batch element, selected on the importance summed over its kv heads (fp32, in
                                                head order) and drawn with the random stream of the call's first head; every
                                                head's out_idx row holds that set and out_K/out_V are gathered with it */
#define NACL_FLAG_SCORE_CUDA_CORES 0x100u    /* debugging: run the generic CUDA-core scoring kernels even where
                                                the tensor-core path applies */
#define NACL_FLAG_SELECT_GENERAL 0x400u      /* debugging / profiling: the selection takes the general three-pass radix path even
                                                where the one-pass bucket path applies (same result, bit for bit) */
#define NACL_FLAG_GATHER_SEPARATE 0x800u     /* debugging / profiling: the K/V gather always runs as a kernel of its own */
#define NACL_FLAG_SELECT_SHARE_SMS 0x1000u   /* the call runs beside other GPU work (nacl_evict_batch sets it): the selection
                                                kernel's grid stays below ~45 % of the SMs */
#define NACL_FLAG_SCORE_TWO_LAUNCHES 0x200u  /* debugging / profiling: the tensor-core path runs its statistics sweep and its
                                                column-sum sweep as two launches instead of one cooperative launch */

typedef struct nacl_params {
  uint32_t struct_size;            /* = sizeof(nacl_params_t) */
  int32_t dtype;                   /* NACL_DTYPE_* of K, V, Qproxy, out_K, out_V */
  const void* K;                   /* [batch,Hkv,L,d] */
  const void* V;                   /* [batch,Hkv,L,d] */
  const void* Qproxy;              /* [batch,Hq,P,d] */
  int32_t batch, L, Hq, Hkv, d, P;
  int32_t budget_proxy, budget_random, n_sink, n_recent;
  uint64_t seed;
  int32_t layer;
  uint32_t flags;
  void* out_K;                     /* [batch,Hkv,C,d] */
  void* out_V;                     /* [batch,Hkv,C,d] */
  int32_t* out_idx;                /* [batch,Hkv,C] */
  float* out_importance;           /* optional [batch,Hkv,L] */
  float* out_lse;                  /* optional [batch,Hq,P]: ln sum_j exp(s[i,j]) */
  void* workspace;                 /* optional; >= nacl_workspace_bytes(...) bytes, 256-byte aligned */
  size_t workspace_bytes;
  void* stream;                    /* cudaStream_t */
  const float* lse_in;             /* optional [batch,Hq,P] fp32: the natural-log row normaliser of every proxy row, as a
                                      prefill attention kernel that keeps its softmax statistics already has it (the contract of
                                      the paper's Algorithm 2).  When given, the statistics sweep over K is
                                      skipped: one logit sweep instead of two.  WHICH normaliser, by flags:
                                        default (no mask, R1): ln sum_{j < L} exp(s[i,j]) over ALL L keys -- a causal
                                          prefill's LSE of row i misses the keys j > L-P+i and is NOT this quantity;
                                        NACL_FLAG_CAUSAL: ln sum_{j <= L-P+i} exp(s[i,j]), exactly what a causal forward pass
                                          stores (Algorithm 2 proper).
                                      The caller answers for its accuracy: imp[j] = sum_i exp(s[i,j] - lse_in[i]). */
  int32_t batch_offset;            /* global index of this call's batch element 0 and ...                                  */
  int32_t head_offset;             /* ... of its kv head 0: the Random Eviction draws are keyed by the GLOBAL (layer, batch,
                                      kv head, position) ("different seed on attention heads and layers"), so a
                                      caller that holds a slice of the heads (tensor parallel) or of the batch (data parallel)
                                      passes where its slice starts and draws exactly what the unsharded call draws.  >= 0;
                                      0 for an unsharded call */
  const int32_t* protect_idx;      /* optional DEVICE array [n_protect]: further protected positions (Table "hyperp",
                                      PAPER.md:490-494: "protect proxy"), strictly ascending, inside [n_sink, L - n_recent), the
                                      same for every batch element and head.  They are always retained and count inside
                                      budget_proxy (R7): budget_proxy >= n_sink + n_recent + n_protect.  The
                                      contents are the caller's responsibility (validation never reads device memory) */
  int32_t n_protect;
  int32_t reserved0;               /* 0 */
  int64_t kv_stride_batch;         /* ELEMENT strides of K and V between batch elements, kv heads and key rows; the d      */
  int64_t kv_stride_head;          /* elements of one row are contiguous.  All three 0 = contiguous [batch,Hkv,L,d].       */
  int64_t kv_stride_row;           /* Otherwise all three > 0, e.g. a cache [batch,Hkv,cap,d] with cap >= L rows per head   */
                                   /* (row = d, head = cap*d, batch = Hkv*cap*d) or a token-major [batch,L,Hkv,d] tensor   */
                                   /* (row = Hkv*d, head = d, batch = L*Hkv*d).  Each times sizeof(element) must be a      */
                                   /* multiple of 16 bytes.  K and V share them ("compatible with            */
                                   /* FlashAttention": both cache layouts of such kernels are served without a copy)       */
  /* In-place compaction: out_K == K and out_V == V with the SAME strides and contiguous rows
     (kv_stride_row == d) compacts the cache inside its own buffers: rows 0 .. C-1 of every head receive the kept rows
     (a row is never overwritten before it has been read), the rows behind them keep their old contents.  Needs the
     cluster selection kernel (rows of at most 327680 keys, not NACL_FLAG_SHARED_HEADS, not paged): NACL_ERR_UNSUPPORTED
     otherwise.  Any other overlap between inputs and outputs is undefined. */
  int64_t out_stride_batch;        /* the same for out_K / out_V; all three 0 = contiguous [batch,Hkv,C,d]                  */
  int64_t out_stride_head;
  int64_t out_stride_row;
  /* Paged K/V (the block-table caches of paged-attention servers): with block_table != NULL, K and V
     are page POOLS and position j of batch element b lives in page block_table[b*table_stride + j/page_size], row
     j % page_size of that page.  kv_stride_page / kv_stride_head / kv_stride_row are the ELEMENT strides between pages,
     between the kv heads of a page and between the rows of a page (all three 0 = a contiguous pool
     [n_pages, Hkv, page_size, d]; kv_stride_batch is ignored).  page_size: 8, 16, 32, 64 or 128.  table_stride >=
     ceil(L / page_size); the entries of the pages that hold positions < L must lie in [0, n_pages) (device memory: not
     validated).  Served by the tensor-core scoring path only (bf16, d = 128, G*P a multiple of 16):
     NACL_ERR_UNSUPPORTED otherwise.  out_K / out_V stay dense. */
  const int32_t* block_table;      /* DEVICE [batch, table_stride] int32, or NULL */
  int32_t page_size;
  int32_t table_stride;
  int32_t n_pages;
  int32_t reserved1;               /* 0 */
  int64_t kv_stride_page;
} nacl_params_t;

/* bf16 K/V/Q.  Steps 1-7 above on `stream`. */
int nacl_evict(const void* K, const void* V, const void* Qproxy,
               int batch, int L, int Hq, int Hkv, int d, int P,
               int budget_proxy, int budget_random, int n_sink, int n_recent,
               uint64_t seed, int layer,
               void* out_K, void* out_V, int32_t* out_idx, void* stream);

/* fp32 K/V/Q, otherwise identical. */
int nacl_evict_f32(const void* K, const void* V, const void* Qproxy,
                   int batch, int L, int Hq, int Hkv, int d, int P,
                   int budget_proxy, int budget_random, int n_sink, int n_recent,
                   uint64_t seed, int layer,
                   void* out_K, void* out_V, int32_t* out_idx, void* stream);

/* Superset entry point: dtype tag, flags, optional importance / lse outputs, explicit workspace. */
int nacl_evict_ex(const nacl_params_t* p);

/* Step 1-2 on their own: the log-sum-exp of every proxy row over the keys (the "LSE emission" half of SURVEY.md 8(f) f4;
 * PAPER.md:507 "The forward computation of FlashAttention-2 returns the log-sum-exp for each row", :518-536 Algorithm 2).
 *   out_lse[b,hq,i] = ln sum_j exp(Q[b,hq,i,:] . K[b,hq/G,j,:] / sqrt(d))      (fp32, [batch,Hq,P]; under NACL_FLAG_CAUSAL the
 *   sum runs over j <= L-P+i)
 * One sweep over K (the statistics sweep of nacl_evict_ex) and a small merge; no importance, no selection, no gather.  It
 * is the producer for nacl_params_t.lse_in when the prefill attention kernel does not hand its softmax statistics out: a
 * caller runs it beside (or right after) its own prefill of the layer and then calls nacl_evict_ex with lse_in = out_lse,
 * which is left with a single sweep.  (Emitting the statistics from inside the prefill attention itself would need that
 * kernel, which is outside this library.)
 * Read from *p: dtype, K, Qproxy, batch, L, Hq, Hkv, d, P, the K strides / block table, flags (NACL_FLAG_CAUSAL,
 * NACL_FLAG_SCORE_CUDA_CORES only), out_lse (required), workspace / workspace_bytes (optional, as for nacl_evict_ex), stream.
 * V, the budgets, protect_idx and the other outputs are ignored; lse_in and out_importance must be NULL. */
int nacl_proxy_lse(const nacl_params_t* p);

/* nacl_evict_ex for callers that must not allocate device memory.
 *
 * Who that is: an inference server that hands (nearly) all of the GPU's memory to its own KV-cache pool at start-up, so
 * that any cudaMalloc afterwards fails or, worse, succeeds by taking memory the pool was promised; a decode loop in
 * which cudaMalloc / cudaFree are unwelcome because they synchronise the whole device and stall every stream; a plug-in
 * or worker whose host application owns the allocator and forbids its guests to go to the driver behind its back.
 * nacl_evict / nacl_evict_ex without a workspace cudaMalloc a per-stream workspace on first use (and again when a larger
 * shape arrives); nacl_evict_ex WITH a workspace allocates nothing but asks the caller for device memory, which such a
 * caller may have no spare byte of.  This entry point needs neither.
 *
 * What it does instead: the scratch the kernels need (softmax partials, the importance rows, hand-over counters; what
 * nacl_workspace_bytes counts) is a fixed array of NACL_STATIC_SCRATCH_BYTES inside the library's device image.  The
 * price is that every GPU on which the library is loaded carries those bytes from load until the process exits, whether
 * or not this function is ever called; 16 MiB holds each of the five BASELINE.json shapes (the largest, batch 4 x 8 kv
 * heads x 32768 keys, needs 14.7 MiB).  The function calls no cudaMalloc, cudaFree, stream / event creation or any other
 * allocating routine (with nacl_profile_enable on, event pairs are created as for every other call: leave it off).
 * K, V, Qproxy and the outputs remain the caller's buffers, exactly as for nacl_evict_ex.
 *
 * Arguments: *p as for nacl_evict_ex, every option included, except that p->workspace must be NULL and
 * p->workspace_bytes 0 (NACL_ERR_WORKSPACE otherwise).  Results are bit-identical to nacl_evict_ex on the same inputs.
 * A shape with nacl_workspace_bytes(batch, L, Hq, Hkv, d, P) > NACL_STATIC_SCRATCH_BYTES is refused with
 * NACL_ERR_STATIC_LIMIT before anything is enqueued or written; that check is host-side and needs no GPU.
 *
 * First call on a device: it looks up where the array lives on the device that is current (one cudaGetSymbolAddress,
 * remembered per device; no memory is obtained by it).  Make that first call, on every device you use, during
 * start-up and before any stream capture begins.
 *
 * Sharing: there is ONE array per GPU and every call of this function on that GPU works in it, whatever its stream
 * and whichever host thread issues it.  Calls that follow each other on one stream are fine: each call clears the few
 * counters that have to start at zero and overwrites the rest before reading it, so the leftovers of an earlier call (of
 * any shape) are harmless.  Calls that can be in flight on the GPU at the same time -- different streams without an
 * event between them, for instance host threads that each use a stream of their own -- race on the array and produce garbage:
 * order them yourself, or use nacl_evict_ex with separate workspaces for the concurrent ones. */
#define NACL_STATIC_SCRATCH_BYTES (16 * 1024 * 1024)
int nacl_evict_static(const nacl_params_t* p);

/* n INDEPENDENT calls (e.g. the layers of one prefill: "one-shot eviction after the encoding phase"), any mix
 * of shapes, all with the same p[i].stream.  The calls alternate between two internal streams that fork from and join into
 * that stream: the scoring of call i+1 fills the SMs that the latency-bound selection and the bandwidth-bound gather of call
 * i leave idle (-5 % at cfg 4, -17..22 % at cfgs 2, 3, 5 against n nacl_evict_ex calls).  Results are identical to n
 * nacl_evict_ex calls.  Calls i and i+1 may run at the same time: caller workspaces (p[i].workspace) of neighbouring calls
 * must not overlap (NULL = the library's own, one per internal stream); outputs of different calls must not overlap either.
 * Capturable into a CUDA graph once the library's streams exist (after one eager call).  Returns the first error. */
int nacl_evict_batch(const nacl_params_t* p, int n);

/* Generation-phase eviction ("Generation Phase Eviction"; Algorithm 1, function Generation):
 * every m decoding steps the cache of a layer, which has grown to `len` = C + m entries per head, is cut back to the budget
 * C = budget_proxy + budget_random by the SAME eviction (Algorithm 1 lines 7-10) driven by the attention row of the current
 * token alone, A_t = q_t K_t^T / sqrt(d) in R^{1 x len}: one proxy row per query head, its softmax over the live cache
 * entries, summed over the G query heads of a kv head.  Cache SLOTS take the place of prompt positions: the first n_sink
 * slots and the last n_recent slots (the newest tokens) are protected.  The draws of the Random Eviction at decoding step
 * `step` use the seed  seed + step * 0x9E3779B97F4A7C15  (independent streams per step; R16).
 *   K_cache, V_cache [batch, Hkv, cap_in, d]   the first `len` rows of every head are live
 *   q                [batch, Hq, 1, d]         the current token's queries
 *   pos_in  (optional) [batch, Hkv, cap_in] int32: original token position of every live slot
 *   K_out, V_out     [batch, Hkv, cap_out, d]  cap_out >= C; rows [0, C) receive the compacted cache (must not alias the inputs)
 *   pos_out (with pos_in) [batch, Hkv, cap_out] int32: pos_out[c] = pos_in[slot kept at c]
 *   out_idx (optional) [batch, Hkv, C] int32: the kept cache slots, ascending
 *   out_importance (optional) [batch, Hkv, len] fp32
 * All DEVICE pointers, same alignment rules, enqueued on `stream`.  It is nacl_evict_ex with P = 1, L = len and the cache's
 * strides, followed by the position-map update. */
typedef struct nacl_gen_params {
  uint32_t struct_size;            /* = sizeof(nacl_gen_params_t) */
  int32_t dtype;
  const void* K_cache;
  const void* V_cache;
  const void* q;
  const int32_t* pos_in;
  int32_t batch, Hq, Hkv, d, len, cap_in, cap_out;
  int32_t budget_proxy, budget_random, n_sink, n_recent;
  uint64_t seed;
  int32_t layer, step;
  uint32_t flags;                  /* NACL_FLAG_SAMPLE_*, NACL_FLAG_SHARED_HEADS, NACL_FLAG_SCORE_CUDA_CORES */
  int32_t batch_offset, head_offset, reserved0;
  void* K_out;
  void* V_out;
  int32_t* pos_out;
  int32_t* out_idx;
  float* out_importance;
  void* workspace;                 /* optional; >= nacl_workspace_bytes(batch, len, Hq, Hkv, d, 1) */
  size_t workspace_bytes;
  void* stream;
} nacl_gen_params_t;
int nacl_evict_generation(const nacl_gen_params_t* g);

/* Variable-length batches ("compatible with FlashAttention": padded / varlen prompt batches).
 * Batch element b holds seq_len[b] <= p->L live keys in the padded K/V [batch, Hkv, p->L, d] (or the strided layout p
 * describes), its proxy queries Qproxy[b] are the last P positions of ITS prompt, and it keeps budget_proxy[b] +
 * budget_random[b] <= C_max positions: rows 0 .. C_b-1 of its slices of out_K / out_V [batch, Hkv, C_max, d] (or the strided
 * output layout of p; rows past C_b are left untouched) and, PACKED as [Hkv, C_b], the first Hkv*C_b entries of its slice
 * out_idx[b*Hkv*C_max ...].  seq_len, budget_proxy, budget_random: HOST arrays of `batch` ints (read before the call
 * returns); p->budget_proxy / p->budget_random are ignored.  Every element is evicted exactly as a batch-1 nacl_evict_ex call
 * with batch_offset = p->batch_offset + b would evict it (same Philox streams), one after the other on p->stream.
 * lse_in, out_importance, out_lse and protect_idx must be NULL.  Every element's length and budgets are validated (as a
 * batch-1 call would: P <= seq_len[b], n_sink + n_recent <= seq_len[b], budget_proxy[b] >= n_sink + n_recent, total <=
 * seq_len[b]) before the first launch, so a validation error writes nothing; an element that keeps nothing
 * (budget_proxy[b] + budget_random[b] == 0) is skipped.  This is a host loop: batch launch sets one after the other, each
 * over Hkv heads only (a padded batch of equal lengths is served faster by one nacl_evict_ex call).  Returns the first
 * error, NACL_OK otherwise. */
int nacl_evict_varlen(const nacl_params_t* p, const int32_t* seq_len, const int32_t* budget_proxy,
                      const int32_t* budget_random, int C_max);

/* Same operation with every tensor in HOST memory (pinned memory makes the copies
 * asynchronous).  Copies K, V, Qproxy to grow-only device staging buffers, runs steps 1-7
 * and copies out_K, out_V, out_idx back; returns after the results are in host memory.
 * device < 0 uses the current device. */
int nacl_evict_host(const void* K, const void* V, const void* Qproxy, int dtype,
                    int batch, int L, int Hq, int Hkv, int d, int P,
                    int budget_proxy, int budget_random, int n_sink, int n_recent,
                    uint64_t seed, int layer,
                    void* out_K, void* out_V, int32_t* out_idx, int device);

/* n problems of ONE shape out of host memory (e.g. the layers of a prefill whose K/V were offloaded): K[i], V[i],
 * Qproxy[i], out_K[i], out_V[i], out_idx[i] are HOST pointers as for nacl_evict_host, seed[i] / layer[i] the problem's seed
 * and layer.  Two staging slots with a stream each: the host-to-device copies of problem i+1 run under the kernels and the
 * device-to-host copies of problem i.  Returns after all results are in host memory. */
int nacl_evict_host_batch(int n, const void* const* K, const void* const* V, const void* const* Qproxy, int dtype,
                          int batch, int L, int Hq, int Hkv, int d, int P,
                          int budget_proxy, int budget_random, int n_sink, int n_recent,
                          const uint64_t* seed, const int32_t* layer,
                          void* const* out_K, void* const* out_V, int32_t* const* out_idx, int device);

/* Step 5 on its own (R4/R5/R10/R15): the Random-Eviction sampling key of EVERY position,
 *   out_keys[b,hk,j] = fl32( ln w_j - ln(-ln u_j) ),  u_j = Philox4x32-10(counter = (j, hk, b, layer), key = seed),
 * w_j = importance[b,hk,j] (or exp / 1 under the NACL_FLAG_SAMPLE_* flags); -inf where w_j = 0.  The budget_random
 * positions with the largest keys among the candidates are the sample.  importance, out_keys: DEVICE pointers,
 * [batch,Hkv,L] fp32, 4-byte aligned; enqueued on `stream`.  nacl_evict computes the same keys internally. */
int nacl_gumbel_keys(const float* importance, float* out_keys, int batch, int Hkv, int L,
                     uint64_t seed, int layer, uint32_t flags, void* stream);

/* Bytes of scratch one call needs (a pure function of the shape; 0 on invalid shapes). */
size_t nacl_workspace_bytes(int batch, int L, int Hq, int Hkv, int d, int P);

/* Per-stage device timing, for benchmarks.  While enabled, every call brackets each of its kernel
 * launches with a pair of CUDA events on the call's stream (so calls are NOT graph-capturable while
 * enabled).  nacl_profile_read waits for the recorded events, adds their elapsed times to per-stage
 * totals and returns the totals accumulated since the last reset: ms[s] = device milliseconds and
 * launches[s] = kernel launches of stage s, s < NACL_N_STAGES (stage names: nacl_stage_name): the way to
 * count what a call really launched (the number depends on shape, flags and on the cluster sizes the device can schedule).
 * Either output may be NULL.  Returns 0 or NACL_ERR_CUDA. */
#define NACL_N_STAGES 7
int nacl_profile_enable(int on);
int nacl_profile_read(double* ms, int64_t* launches, int reset);
const char* nacl_stage_name(int stage);

/* Diagnostics: the number of (batch, kv head) selections on the current device that left the one-pass bucket path for the
 * general three-pass radix path since the last reset (a threshold in a clamped edge bucket, a candidate list that
 * would overflow; the result is the same either way).  Synchronises the device.  Returns the count or NACL_ERR_CUDA. */
int nacl_select_fallbacks(int reset);

/* Diagnostics: the launch configuration of the selection kernel that the latest eviction call ISSUED FROM THIS HOST THREAD
 * chose: CTAs in its grid, CTAs per cluster (0 = the path without clusters, one CTA per head) and whether that kernel also
 * moved the kept K/V rows (1) or a stand-alone gather followed (0).  Lets a test or a benchmark assert which launch
 * configuration it really ran (e.g. nacl_evict_batch keeps the grid below ~45 % of the SMs).  Outputs may be NULL. */
void nacl_last_select_launch(int* grid_ctas, int* cluster_size, int* fused_gather);

/* Frees the per-device internal workspaces / staging buffers (optional, e.g. before exit). */
void nacl_release(void);

const char* nacl_strerror(int code);
/* cudaError_t of the most recent NACL_ERR_CUDA on this thread, as an int. */
int nacl_last_cuda_error(void);
int nacl_version(void);

#ifdef __cplusplus
}
#endif
#endif
