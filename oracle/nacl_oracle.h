/*
 * nacl_oracle.h -- CPU ORACLE for NACL one-shot encoding-phase KV-cache eviction
 * (arXiv 2408.03675).  THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, fp64, step-by-step restatement of what the paper defines
 * (PAPER.md = /root/reference/PAPER.md, cited by line; readings R1..R15 are
 * listed in DESIGN.md).  It shares no code with the CUDA path under
 * paper_2408_03675_b200/csrc and neither side includes or links the other.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may call it.
 *
 * Parity status: every function below is pinned by tests/test_oracle_*.py
 * against values the paper / mathematics fix, except
 *   - "which indices a given seed must draw on the large configs": PARITY
 *     UNPINNED beyond the Philox known-answer vectors, the sampling-law
 *     chi-square/enumeration tests on tiny inputs and determinism; no external
 *     reference exists for those values, the oracle defines them.
 *
 * All pointers are HOST pointers.  Layouts are contiguous row-major:
 *   K, V   : [batch, Hkv, L, d]        Q : [batch, Hq, P, d]  (the P proxy rows
 *            are the queries of the last P prompt positions, in order)
 *   imp    : [batch, Hkv, L] fp64      lse : [batch, Hq, P] fp64
 *   out_idx: [batch, Hkv, C] int32, C = budget_proxy + budget_random
 * dtype: 0 = IEEE fp32, 1 = bfloat16 (upper 16 bits of an fp32).
 * Every function returns 0 on success, a negative NACL_ORACLE_E* otherwise.
 */
#ifndef NACL_ORACLE_H
#define NACL_ORACLE_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define NACL_ORACLE_F32 0
#define NACL_ORACLE_BF16 1

/* flags (readings R1, R4) */
#define NACL_ORACLE_CAUSAL 1u                 /* row i (position L-P+i) sees keys j <= L-P+i */
#define NACL_ORACLE_SAMPLE_SOFTMAX_OF_SCORE 2u /* weights exp(imp_j) instead of imp_j */
#define NACL_ORACLE_SAMPLE_UNIFORM 4u          /* uniform weights (paper's ablation) */

#define NACL_ORACLE_EARG (-1)
#define NACL_ORACLE_EBUDGET (-2)
#define NACL_ORACLE_ENOMEM (-3)

/* Philox4x32-10, Salmon et al. SC'11 (R10). */
void nacl_oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);

/* u in (0,1) for (seed, layer, batch b, kv head hk, position j):
 * word 0 of Philox(ctr=(j,hk,b,layer), key=(lo32 seed, hi32 seed)),
 * u = ((x >> 9) + 0.5) * 2^-23.  ("different seed on attention
 * heads and layers"; R10) */
double nacl_oracle_uniform(uint64_t seed, int layer, int b, int hk, int j);

/* Gumbel-top-k key of one candidate (R4, R5):
 * fl32( ln(w) - ln(-ln u) ), evaluated in fp64 and rounded once to fp32 (the
 * precision in which both sides take the selection decision).  w = imp,
 * exp(imp) or 1 according to flags; w = 0 gives -inf. */
float nacl_oracle_gumbel_key(double imp, double u, unsigned flags);

/* Steps 1-3: logits, row softmax, column sum. */
int nacl_oracle_importance(const void* K, const void* Q, int dtype,
                           int batch, int L, int Hq, int Hkv, int d, int P,
                           unsigned flags, double* imp, double* lse /*nullable*/, int nthreads);

/* Steps 4-7: protected set, top-k, Gumbel-top-k sample, ascending merge
 * (PAPER.md:134-140, 148-163, 179-183).
 * out_part  (nullable) [batch,Hkv,C]: 0 = protected, 1 = top-k, 2 = random.
 * out_key   (nullable) [batch,Hkv,L]: the fp32 sampling key of every candidate
 *           of the random stage, NaN for non-candidates. */
int nacl_oracle_select(const double* imp, int batch, int L, int Hkv,
                       int budget_proxy, int budget_random, int n_sink, int n_recent,
                       uint64_t seed, int layer, unsigned flags,
                       int32_t* out_idx, int32_t* out_part, float* out_key);

/* Steps 4-7 with the options the paper's variants need (NULL opts = nacl_oracle_select):
 *   batch_offset, head_offset: GLOBAL index of batch element 0 / kv head 0 of this call in the Philox counter (R10;
 *       PAPER.md:37 ties the stream to the head and the layer, not to the device that holds it), so that a shard of the
 *       heads or of the batch draws exactly what the unsharded problem draws;
 *   protect_idx[n_protect]: further protected positions, ascending, unique, inside [n_sink, L - n_recent), the same for
 *       every problem (Table "hyperp": "protect proxy"); they count inside budget_proxy (R7);
 *   shared_heads != 0: the "- Head-wise" ablation: one retained set per batch element, chosen
 *       on the importance summed over the kv heads, drawn with the stream of the call's first head. */
typedef struct {
  int batch_offset, head_offset;
  const int32_t* protect_idx;
  int n_protect;
  int shared_heads;
} nacl_oracle_select_opts;
int nacl_oracle_select_ex(const double* imp, int batch, int L, int Hkv,
                          int budget_proxy, int budget_random, int n_sink, int n_recent,
                          uint64_t seed, int layer, unsigned flags, const nacl_oracle_select_opts* opts,
                          int32_t* out_idx, int32_t* out_part, float* out_key);

/* Step 8: K,V <- K_S,V_S by copying the original bytes. */
int nacl_oracle_gather(const void* K, const void* V, size_t row_bytes,
                       int batch, int L, int Hkv, int C, const int32_t* idx,
                       void* out_K, void* out_V);

/* Steps 1-8. out_imp (nullable) [batch,Hkv,L] fp64. */
int nacl_oracle_evict(const void* K, const void* V, const void* Q, int dtype,
                      int batch, int L, int Hq, int Hkv, int d, int P,
                      int budget_proxy, int budget_random, int n_sink, int n_recent,
                      uint64_t seed, int layer, unsigned flags,
                      void* out_K, void* out_V, int32_t* out_idx,
                      double* out_imp, int nthreads);

/* number of OpenMP threads a call with this nthreads argument will use */
int nacl_oracle_threads(int nthreads);

#ifdef __cplusplus
}
#endif
#endif
