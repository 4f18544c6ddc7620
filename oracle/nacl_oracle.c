/*
 * nacl_oracle.c -- CPU ORACLE (test infrastructure, not the product) for
 * NACL one-shot encoding-phase KV-cache eviction, arXiv 2408.03675.
 *
 * Plain C, fp64, no blocking / fusion / reordering beyond what the paper's
 * definitions state.  See nacl_oracle.h for the contract and DESIGN.md for the
 * readings (R1..R15) taken where PAPER.md is silent or garbled.  This file
 * shares nothing with the CUDA path.
 *
 * Build: gcc -O2 -std=c11 -fopenmp -fPIC -shared nacl_oracle.c -lm
 * (no -ffast-math: the arithmetic order below is the one written).
 */
#include "nacl_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ------------------------------------------------------------------ helpers */

int nacl_oracle_threads(int nthreads) {
#ifdef _OPENMP
  return nthreads > 0 ? nthreads : omp_get_max_threads();
#else
  (void)nthreads;
  return 1;
#endif
}

/* exact widening of one stored element to fp64 */
static double load_elem(const void* base, size_t idx, int dtype) {
  if (dtype == NACL_ORACLE_F32) {
    return (double)((const float*)base)[idx];
  } else { /* bfloat16 = the upper 16 bits of an IEEE fp32 */
    uint32_t bits = ((uint32_t)((const uint16_t*)base)[idx]) << 16;
    float f;
    memcpy(&f, &bits, sizeof f);
    return (double)f;
  }
}

/* ------------------------------------------------------- Philox4x32-10 (R10) */
/* Salmon, Moraes, Dror, Shaw: "Parallel random numbers: as easy as 1, 2, 3",
 * SC'11.  One round: (c0,c1,c2,c3) <- (hi(M1*c2)^c1^k0, lo(M1*c2),
 * hi(M0*c0)^c3^k1, lo(M0*c0)); then the key is bumped by the Weyl constants. */
void nacl_oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
  const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    uint64_t p0 = (uint64_t)M0 * c0;
    uint64_t p1 = (uint64_t)M1 * c2;
    uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    uint32_t n0 = hi1 ^ c1 ^ k0;
    uint32_t n1 = lo1;
    uint32_t n2 = hi0 ^ c3 ^ k1;
    uint32_t n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += W0; k1 += W1;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* PAPER.md:37 ("different seed on attention heads and layers"); R10:
 * counter = (position, kv head, batch, layer), key = the 64-bit seed. */
double nacl_oracle_uniform(uint64_t seed, int layer, int b, int hk, int j) {
  uint32_t ctr[4] = {(uint32_t)j, (uint32_t)hk, (uint32_t)b, (uint32_t)layer};
  uint32_t key[2] = {(uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32)};
  uint32_t x[4];
  nacl_oracle_philox4x32_10(ctr, key, x);
  /* 23 bits, centred: u in [2^-24, 1-2^-24], exactly representable in fp32 and fp64 */
  return ((double)(x[0] >> 9) + 0.5) * 0x1p-23;
}

/* PAPER.md:150-161 (Random Eviction): S_random ~ P_prompt, |S_random| = C_r,
 * "P_random can be based on the normalized distribution Softmax(F_score)".
 * DESIGN.md R4: probability proportional to importance; R5: sampling without
 * replacement with renormalisation after each draw == Gumbel-top-k: perturb
 * ln(weight) with i.i.d. Gumbel noise -ln(-ln u) and keep the largest C_r. */
float nacl_oracle_gumbel_key(double imp, double u, unsigned flags) {
  double ln_w;
  if (flags & NACL_ORACLE_SAMPLE_UNIFORM) {
    ln_w = 0.0;
  } else if (flags & NACL_ORACLE_SAMPLE_SOFTMAX_OF_SCORE) {
    ln_w = imp; /* weight exp(imp) */
  } else {
    ln_w = log(imp); /* weight imp; imp = 0 -> -inf (R13) */
  }
  double gumbel = -log(-log(u));
  return (float)(ln_w + gumbel); /* one rounding, fp64 -> fp32 */
}

/* --------------------------------------------- steps 1-3: importance scores */
int nacl_oracle_importance(const void* K, const void* Q, int dtype,
                           int batch, int L, int Hq, int Hkv, int d, int P,
                           unsigned flags, double* imp, double* lse, int nthreads) {
  if (!K || !Q || !imp) return NACL_ORACLE_EARG;
  if (dtype != NACL_ORACLE_F32 && dtype != NACL_ORACLE_BF16) return NACL_ORACLE_EARG;
  if (batch < 1 || L < 1 || Hq < 1 || Hkv < 1 || d < 1 || P < 1 || P > L) return NACL_ORACLE_EARG;
  if (Hq % Hkv != 0) return NACL_ORACLE_EARG;
  const int G = Hq / Hkv; /* R3: query head hq reads kv head hq / G */
  const int rows = G * P;
  const int causal = (flags & NACL_ORACLE_CAUSAL) != 0;
  const int nt = nacl_oracle_threads(nthreads);
  (void)nt;

  double* Kd = (double*)malloc((size_t)L * d * sizeof(double));
  double* Qd = (double*)malloc((size_t)rows * d * sizeof(double));
  double* prob = (double*)malloc((size_t)rows * L * sizeof(double)); /* Softmax(A(x_p,*)), all proxy rows */
  if (!Kd || !Qd || !prob) { free(Kd); free(Qd); free(prob); return NACL_ORACLE_ENOMEM; }
  const double inv_sqrt_d = 1.0 / sqrt((double)d); /* R2: 1/sqrt(head_dim) */

  for (int b = 0; b < batch; ++b) {
    for (int hk = 0; hk < Hkv; ++hk) {
      const size_t kbase = ((size_t)b * Hkv + hk) * (size_t)L * d;
      for (size_t e = 0; e < (size_t)L * d; ++e) Kd[e] = load_elem(K, kbase + e, dtype);
      for (int g = 0; g < G; ++g) {
        const int hq = hk * G + g;
        const size_t qbase = ((size_t)b * Hq + hq) * (size_t)P * d;
        for (size_t e = 0; e < (size_t)P * d; ++e) Qd[(size_t)g * P * d + e] = load_elem(Q, qbase + e, dtype);
      }

      /* one proxy row at a time: A(x_p,*) then Softmax */
#pragma omp parallel for schedule(dynamic, 1) num_threads(nt)
      for (int r = 0; r < rows; ++r) {
        const int i = r % P;                        /* proxy row i is prompt position L-P+i */
        const int last_visible = causal ? (L - P + i) : (L - 1);
        const double* q = Qd + (size_t)r * d;
        double* p = prob + (size_t)r * L;
        double m = -INFINITY;
        for (int j = 0; j <= last_visible; ++j) {
          const double* k = Kd + (size_t)j * d;
          double dot = 0.0;
          for (int t = 0; t < d; ++t) dot += q[t] * k[t];
          p[j] = dot * inv_sqrt_d;                   /* logit A(x_p, j) */
          if (p[j] > m) m = p[j];
        }
        double Z = 0.0;
        for (int j = 0; j <= last_visible; ++j) Z += exp(p[j] - m);
        for (int j = 0; j <= last_visible; ++j) p[j] = exp(p[j] - m) / Z;
        for (int j = last_visible + 1; j < L; ++j) p[j] = 0.0; /* masked */
        if (lse) {
          const int g = r / P;
          lse[((size_t)b * Hq + (hk * G + g)) * P + i] = m + log(Z);
        }
      }

      /* F_score = sum over proxy rows (and over the GQA group, R3), fixed row order */
      double* out = imp + ((size_t)b * Hkv + hk) * (size_t)L;
#pragma omp parallel for schedule(static) num_threads(nt)
      for (int j = 0; j < L; ++j) {
        double acc = 0.0;
        for (int r = 0; r < rows; ++r) acc += prob[(size_t)r * L + j];
        out[j] = acc;
      }
    }
  }
  free(Kd); free(Qd); free(prob);
  return 0;
}

/* ------------------------------------------------- steps 4-7: the index set */
typedef struct { double v; int32_t j; } score_item;
typedef struct { float v; int32_t j; } key_item;

/* (value descending, index ascending): ties go to the lower index (R9) */
static int cmp_score_desc(const void* a, const void* b) {
  const score_item* x = (const score_item*)a;
  const score_item* y = (const score_item*)b;
  if (x->v > y->v) return -1;
  if (x->v < y->v) return 1;
  return (x->j > y->j) - (x->j < y->j);
}
static int cmp_key_desc(const void* a, const void* b) {
  const key_item* x = (const key_item*)a;
  const key_item* y = (const key_item*)b;
  if (x->v > y->v) return -1;
  if (x->v < y->v) return 1;
  return (x->j > y->j) - (x->j < y->j);
}

/* Steps 4-7 for one problem: s[L] importance, (b_glob, hk_glob) = the GLOBAL batch / kv-head indices that key the
 * random draws (R10), extra[] = n_extra further protected positions.  Writes C indices (and parts / keys). */
static int select_one(const double* s, int L, int budget_proxy, int budget_random, int n_sink, int n_recent,
                      const int32_t* extra, int n_extra, uint64_t seed, int layer, int b_glob, int hk_glob,
                      unsigned flags, score_item* sc, key_item* ky, int8_t* part,
                      int32_t* out_idx, int32_t* out_part, float* out_key) {
  const int C = budget_proxy + budget_random;
  const int lo = n_sink, hi = L - n_recent; /* positions [lo, hi) are not protected by the sink / recent rule */
  for (int j = 0; j < L; ++j)
    if (!(s[j] >= 0.0) || isinf(s[j])) return NACL_ORACLE_EARG; /* importance is a finite sum of probabilities */
  memset(part, -1, (size_t)L);

  /* step 4: protected set Pi = sinks and recent tokens (PAPER.md:137-140 "cup P", :390), plus the explicit list
   * (Table "hyperp": protected proxy tokens count inside the proxy budget, R7) */
  for (int j = 0; j < n_sink; ++j) part[j] = 0;
  for (int j = hi; j < L; ++j) part[j] = 0;
  for (int e = 0; e < n_extra; ++e) {
    const int j = extra[e];
    if (j < lo || j >= hi || (e > 0 && extra[e - 1] >= j)) return NACL_ORACLE_EARG; /* ascending, unique, not already protected */
    part[j] = 0;
  }
  const int k1 = budget_proxy - n_sink - n_recent - n_extra; /* free top-k slots (R7) */
  if (k1 < 0) return NACL_ORACLE_EBUDGET;

  /* step 5: argmax_{S subset R, |S| = C_p} sum F_score: full sort, take the head */
  int n_free = 0;
  for (int j = lo; j < hi; ++j)
    if (part[j] < 0) { sc[n_free].v = s[j]; sc[n_free].j = j; ++n_free; }
  qsort(sc, (size_t)n_free, sizeof(score_item), cmp_score_desc);
  for (int r = 0; r < k1; ++r) part[sc[r].j] = 1;

  /* step 6: Random Eviction over the rest (R4, R5, R6) */
  const int n_cand = n_free - k1;
  if (out_key)
    for (int j = 0; j < L; ++j) out_key[j] = NAN;
  for (int r = 0; r < n_cand; ++r) {
    const int j = sc[k1 + r].j;
    const double u = nacl_oracle_uniform(seed, layer, b_glob, hk_glob, j);
    ky[r].v = nacl_oracle_gumbel_key(s[j], u, flags);
    ky[r].j = j;
    if (out_key) out_key[j] = ky[r].v;
  }
  qsort(ky, (size_t)n_cand, sizeof(key_item), cmp_key_desc);
  for (int r = 0; r < budget_random; ++r) part[ky[r].j] = 2;

  /* step 7: S = u_score cup u_random, ascending */
  int c = 0;
  for (int j = 0; j < L; ++j) {
    if (part[j] >= 0) {
      if (c < C) {
        out_idx[c] = j;
        if (out_part) out_part[c] = part[j];
      }
      ++c;
    }
  }
  return c == C ? 0 : NACL_ORACLE_EARG; /* cannot fail: parts are disjoint by construction */
}

int nacl_oracle_select_ex(const double* imp, int batch, int L, int Hkv,
                          int budget_proxy, int budget_random, int n_sink, int n_recent,
                          uint64_t seed, int layer, unsigned flags, const nacl_oracle_select_opts* opts,
                          int32_t* out_idx, int32_t* out_part, float* out_key) {
  if (!imp || !out_idx) return NACL_ORACLE_EARG;
  if (batch < 1 || L < 1 || Hkv < 1) return NACL_ORACLE_EARG;
  if (n_sink < 0 || n_recent < 0 || budget_proxy < 0 || budget_random < 0) return NACL_ORACLE_EBUDGET;
  const int b_off = opts ? opts->batch_offset : 0, h_off = opts ? opts->head_offset : 0;
  const int n_extra = opts ? opts->n_protect : 0;
  const int32_t* extra = opts ? opts->protect_idx : NULL;
  const int shared = opts ? opts->shared_heads : 0;
  if (b_off < 0 || h_off < 0 || n_extra < 0 || (n_extra > 0 && !extra)) return NACL_ORACLE_EARG;
  const long n_prot = (long)n_sink + n_recent;
  if (n_prot > L) return NACL_ORACLE_EBUDGET;
  if (budget_proxy < n_prot + n_extra) return NACL_ORACLE_EBUDGET;               /* R7 */
  if ((long)budget_proxy + budget_random > L) return NACL_ORACLE_EBUDGET;
  const int C = budget_proxy + budget_random;

  score_item* sc = (score_item*)malloc((size_t)L * sizeof(score_item));
  key_item* ky = (key_item*)malloc((size_t)L * sizeof(key_item));
  int8_t* part = (int8_t*)malloc((size_t)L);
  double* sum = shared ? (double*)malloc((size_t)L * sizeof(double)) : NULL;
  if (!sc || !ky || !part || (shared && !sum)) { free(sc); free(ky); free(part); free(sum); return NACL_ORACLE_ENOMEM; }

  int rc = 0;
  for (int b = 0; b < batch && rc == 0; ++b) {
    if (shared) {
      /* the "- Head-wise" ablation (PAPER.md:319-321 Table 3, :376-380): ONE retained set per batch element, chosen on
       * the importance summed over the kv heads in head order, drawn with the first head's stream, copied to every head */
      for (int j = 0; j < L; ++j) {
        double a = 0.0;
        for (int hk = 0; hk < Hkv; ++hk) a += imp[((size_t)b * Hkv + hk) * (size_t)L + j];
        sum[j] = a;
      }
      const size_t p0 = (size_t)b * Hkv;
      rc = select_one(sum, L, budget_proxy, budget_random, n_sink, n_recent, extra, n_extra, seed, layer, b + b_off, h_off,
                      flags, sc, ky, part, out_idx + p0 * (size_t)C, out_part ? out_part + p0 * (size_t)C : NULL,
                      out_key ? out_key + p0 * (size_t)L : NULL);
      for (int hk = 1; hk < Hkv && rc == 0; ++hk) {
        memcpy(out_idx + (p0 + hk) * (size_t)C, out_idx + p0 * (size_t)C, (size_t)C * sizeof(int32_t));
        if (out_part) memcpy(out_part + (p0 + hk) * (size_t)C, out_part + p0 * (size_t)C, (size_t)C * sizeof(int32_t));
        if (out_key) memcpy(out_key + (p0 + hk) * (size_t)L, out_key + p0 * (size_t)L, (size_t)L * sizeof(float));
      }
      continue;
    }
    for (int hk = 0; hk < Hkv && rc == 0; ++hk) {
      const size_t prob_id = (size_t)b * Hkv + hk;
      rc = select_one(imp + prob_id * (size_t)L, L, budget_proxy, budget_random, n_sink, n_recent, extra, n_extra, seed, layer,
                      b + b_off, hk + h_off, flags, sc, ky, part, out_idx + prob_id * (size_t)C,
                      out_part ? out_part + prob_id * (size_t)C : NULL, out_key ? out_key + prob_id * (size_t)L : NULL);
    }
  }
  free(sc); free(ky); free(part); free(sum);
  return rc;
}

int nacl_oracle_select(const double* imp, int batch, int L, int Hkv,
                       int budget_proxy, int budget_random, int n_sink, int n_recent,
                       uint64_t seed, int layer, unsigned flags,
                       int32_t* out_idx, int32_t* out_part, float* out_key) {
  return nacl_oracle_select_ex(imp, batch, L, Hkv, budget_proxy, budget_random, n_sink, n_recent, seed, layer, flags, NULL,
                               out_idx, out_part, out_key);
}

/* ----------------------------------------------------- step 8: K,V <- K_S,V_S */
int nacl_oracle_gather(const void* K, const void* V, size_t row_bytes,
                       int batch, int L, int Hkv, int C, const int32_t* idx,
                       void* out_K, void* out_V) {
  if (!K || !V || !idx || !out_K || !out_V) return NACL_ORACLE_EARG;
  for (int b = 0; b < batch; ++b)
    for (int hk = 0; hk < Hkv; ++hk) {
      const size_t p = (size_t)b * Hkv + hk;
      for (int c = 0; c < C; ++c) {
        const int32_t j = idx[p * (size_t)C + c];
        if (j < 0 || j >= L) return NACL_ORACLE_EARG;
        const size_t src = (p * (size_t)L + (size_t)j) * row_bytes;
        const size_t dst = (p * (size_t)C + (size_t)c) * row_bytes;
        memcpy((char*)out_K + dst, (const char*)K + src, row_bytes);
        memcpy((char*)out_V + dst, (const char*)V + src, row_bytes);
      }
    }
  return 0;
}

/* ------------------------------------------------------------- steps 1-8 */
int nacl_oracle_evict(const void* K, const void* V, const void* Q, int dtype,
                      int batch, int L, int Hq, int Hkv, int d, int P,
                      int budget_proxy, int budget_random, int n_sink, int n_recent,
                      uint64_t seed, int layer, unsigned flags,
                      void* out_K, void* out_V, int32_t* out_idx,
                      double* out_imp, int nthreads) {
  if (!K || !V || !Q || !out_K || !out_V || !out_idx) return NACL_ORACLE_EARG;
  if (batch < 1 || L < 1 || Hkv < 1) return NACL_ORACLE_EARG;
  double* imp = out_imp;
  if (!imp) {
    imp = (double*)malloc((size_t)batch * Hkv * (size_t)L * sizeof(double));
    if (!imp) return NACL_ORACLE_ENOMEM;
  }
  int rc = nacl_oracle_importance(K, Q, dtype, batch, L, Hq, Hkv, d, P, flags, imp, NULL, nthreads);
  if (rc == 0)
    rc = nacl_oracle_select(imp, batch, L, Hkv, budget_proxy, budget_random, n_sink, n_recent,
                            seed, layer, flags, out_idx, NULL, NULL);
  if (rc == 0) {
    const size_t esz = dtype == NACL_ORACLE_F32 ? 4 : 2;
    rc = nacl_oracle_gather(K, V, (size_t)d * esz, batch, L, Hkv, budget_proxy + budget_random,
                            out_idx, out_K, out_V);
  }
  if (!out_imp) free(imp);
  return rc;
}
