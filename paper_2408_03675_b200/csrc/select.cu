// select.cu -- steps a4-a6 of SURVEY.md section 8: protected set, Proxy-Tokens top-k, Random
// Eviction as Gumbel-top-k, and the ascending kept-position list.
//
//   nacl_keys_kernel  : key[j] = ordermap(fl32(ln w_j - ln(-ln u_j))),  u_j from Philox4x32-10 keyed by
//                  (seed; layer, batch, kv head, position)                PAPER.md:148-161, 37; R4/R5/R10/R15
//   nacl_select_kernel: one CTA per (batch, kv head).  MSB radix select (12+10+10 bits) of the
//                  (budget_proxy - |Pi|) largest importances outside Pi, a second
//                  radix select of the budget_random largest keys among the rest, ties to the lower
//                  index in both (R9), then an order-preserving compaction that emits the
//                  kept positions already ascending -- no sort.
//   nacl_select_cluster_kernel: the same selection with one thread-block CLUSTER (1..16 CTAs) per (batch, kv head), the
//                  CTAs exchanging histogram sums and candidate lists through distributed shared memory.  Default: the
//                  one-pass bucket path (select_fast: one cluster-wide histogram per select over buckets that are fine
//                  where the threshold lies, fp32 key estimates, exact fp64 keys only next to the threshold, exact finish
//                  on a small candidate list); the three-pass radix path on exact keys is the cluster-uniform fallback.
//                  The kernel also moves the kept K/V rows (step a7), in place if asked.
// Integer work only after the keys: results are bit-exact functions of (imp, key).
#include <cooperative_groups.h>
#include <mutex>
#include <math.h>
#include <string.h>

#include "nacl_internal.cuh"

namespace cg = cooperative_groups;

namespace nacl {
namespace {

// ------------------------------------------------------------------ Philox4x32-10
// Salmon et al., SC'11.  Round: (c0,c1,c2,c3) <- (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0)).
__device__ __forceinline__ uint32_t philox4x32_10_word0(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                                        uint32_t k0, uint32_t k1) {
  constexpr uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint64_t p0 = (uint64_t)M0 * c0, p1 = (uint64_t)M1 * c2;  // one 32x32->64 multiply each (IMAD.WIDE)
    const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0, hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    c0 = hi1 ^ c1 ^ k0;
    c1 = lo1;
    c2 = hi0 ^ c3 ^ k1;
    c3 = lo0;
    k0 += W0;
    k1 += W1;
  }
  return c0;
}

// larger float <=> larger uint32 (-inf lowest, +inf highest)
__device__ __forceinline__ uint32_t ordermap(uint32_t bits) {
  return (bits & 0x80000000u) ? ~bits : (bits | 0x80000000u);
}

// ------------------------------------------------------------------ natural logarithm in fp64, table driven
// ln x for finite normal x > 0:  x = 2^e * m, m in (181/256, 181/128];  c = k/128 the nearest multiple of 1/128;
// r = (m - c)/c (|r| <= 5.6e-3; m - c is exact, 1/c tabulated);  ln x = e*ln2 + ln c + log1p(r), ln c and ln 2 as hi + lo
// pairs, log1p by its degree-7 Taylor polynomial (truncation < 2e-19).  About 15 fp64 operations instead of the ~50 of the
// library routine (the sampling keys are fp64-throughput-bound), error ~1 ulp; around x = 1 (c = 1, ln c = 0 exactly)
// the result keeps full RELATIVE accuracy, which -ln u needs for u next to 1.
// table of {1/c, hi(ln c), lo(ln c)}, c = k/128, k = 90..181: csrc/logtab.inc, written by csrc/gen_logtab.py
__device__ const double kLogTab[92][3] = {
#include "logtab.inc"
};
constexpr double kLn2Hi = 0x1.62e42fefa39efp-1, kLn2Lo = 0x1.abc9e3b39803fp-56;
// int <-> double without the conversion unit (the sampling keys are issue- and XU-bound): 2^52 + 2^31 + e has e's two's
// complement in its low word; x + 1.5*2^52 has round-to-nearest-even(x) in its low word.  Both exact.
__device__ __forceinline__ double small_int_to_double(int e) {
  return __hiloint2double(0x43300000, (int)(0x80000000u ^ (uint32_t)e)) - 4503601774854144.0;  // 2^52 + 2^31
}
__device__ __forceinline__ double log_tab(double x) {
  const int hi = __double2hiint(x);
  int e = ((hi >> 20) & 0x7FF) - 1023;
  double m = __hiloint2double((hi & 0x000FFFFF) | 0x3FF00000, __double2loint(x));  // [1, 2)
  if (m > 1.4140625) { m *= 0.5; e += 1; }
  const double kt = fma(m, 128.0, 6755399441055744.0);  // 1.5 * 2^52: k = rn(m * 128) = 90 .. 181 in the low word
  const int k = __double2loint(kt);
  const double kd = kt - 6755399441055744.0;            // (double)k
  const double* t = kLogTab[k - 90];
  const double r = (m - kd * 0.0078125) * __ldg(&t[0]);
  double q = fma(r, 1.0 / 7.0, -1.0 / 6.0);
  q = fma(q, r, 0.2);
  q = fma(q, r, -0.25);
  q = fma(q, r, 1.0 / 3.0);
  q = fma(q, r, -0.5);
  q = q * r * r;
  const double de = small_int_to_double(e);
  return fma(de, kLn2Hi, __ldg(&t[1]) + (r + (q + fma(de, kLn2Lo, __ldg(&t[2])))));
}

// order-mapped Gumbel-top-k key of position j of kv head hk of batch element b (R4/R5/R10/R13/R15)
template <bool ORDERMAP = true>
__device__ __forceinline__ uint32_t gumbel_key(float imp, uint32_t j, uint32_t hk, uint32_t b, uint32_t layer, uint32_t k0, uint32_t k1,
                                               uint32_t flags) {
  const uint32_t x = philox4x32_10_word0(j, hk, b, layer, k0, k1);
  // u = ((x >> 9) + 0.5) * 2^-23, exact, in [2^-24, 1 - 2^-24]: 2^52 + n has n in its low word; 2^52 - 0.5 is a double
  const double u = (__hiloint2double(0x43300000, (int)(x >> 9)) - 4503599627370495.5) * 0x1p-23;
  const double w = (double)imp;
  double ln_w;
  if (flags & NACL_FLAG_SAMPLE_UNIFORM) ln_w = 0.0;
  else if (flags & NACL_FLAG_SAMPLE_SOFTMAX_OF_SCORE) ln_w = w;
  else ln_w = w > 0.0 ? log_tab(w) : -INFINITY;  // w == 0 -> -inf (R13); fp32 subnormals are normal doubles
  const double gumbel = -log_tab(-log_tab(u));
  float f = (float)(ln_w + gumbel);  // one rounding fp64 -> fp32 (R15)
  f += 0.0f;                         // -0 -> +0 so that equal floats have equal bit patterns
  return ORDERMAP ? ordermap(__float_as_uint(f)) : __float_as_uint(f);
}


// fp32 estimate of the same key (not order-mapped), |estimate - key| < 1e-3 whenever the key is finite and its weight
// is a normal float (a subnormal or zero weight gives -inf; the exact key is then below -80 or -inf).  Used by the
// fast selection path to put the candidates into buckets; every decision near the threshold is re-taken on the exact key.
//   -ln u: for u > 63/64 from the series of -log1p(-(1-u)) (1-u is exact), else from lg2.approx (absolute error 2^-22 on
//   (0.5, 2), relative 2^-22 elsewhere): relative error < 4e-5;  -ln(-ln u) and ln w the same way: absolute error < 2e-4.
__device__ __forceinline__ float lg2_approx(float x) {
  float y;
  asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float gumbel_key_estimate(float imp, uint32_t j, uint32_t hk, uint32_t b, uint32_t layer, uint32_t k0,
                                                      uint32_t k1, uint32_t flags) {
  const uint32_t x = philox4x32_10_word0(j, hk, b, layer, k0, k1);
  const float n = __uint_as_float(0x4B000000u | (x >> 9)) - 8388608.0f;  // (float)(x >> 9), exact
  const float u = (n + 0.5f) * 0x1p-23f;                                  // exact (24 significant bits)
  const float v = 1.0f - u;                                               // exact for u >= 0.5
  float a;                                                                // -ln u
  if (v < 0.015625f) a = v * fmaf(v, fmaf(v, fmaf(v, 0.25f, 0.33333334f), 0.5f), 1.0f);
  else a = -0.69314718f * lg2_approx(u);
  const float g = -0.69314718f * lg2_approx(a);
  float ln_w;
  if (flags & NACL_FLAG_SAMPLE_UNIFORM) ln_w = 0.0f;
  else if (flags & NACL_FLAG_SAMPLE_SOFTMAX_OF_SCORE) ln_w = imp;
  else ln_w = 0.69314718f * lg2_approx(imp);  // imp == 0 (or subnormal: flushed) -> -inf
  return ln_w + g;
}

template <bool ORDERMAP>
__global__ void __launch_bounds__(256) nacl_keys_kernel(const float* __restrict__ imp, uint32_t* __restrict__ key,
                                                    int Hkv, int L, uint32_t k0, uint32_t k1, uint32_t layer, uint32_t flags,
                                                    uint32_t b_off, uint32_t h_off) {
  const int p = blockIdx.y;  // b * Hkv + hk
  const int b = p / Hkv, hk = p - b * Hkv;
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= L) return;
  const size_t o = (size_t)p * L + j;
  key[o] = gumbel_key<ORDERMAP>(imp[o], (uint32_t)j, (uint32_t)hk + h_off, (uint32_t)b + b_off, layer, k0, k1, flags);
}

// ------------------------------------------------------------------ block primitives
constexpr int ST = 1024;  // threads of the select CTA
constexpr int HB = 4096;  // histogram bins (12-bit first digit)

struct SelShared {
  uint32_t hist[HB];
  int warp_tot[32];
  int total;
  int bin, krem, lcut;
};

// exclusive prefix sum of v over the block in thread order; total in `tot` (uniform)
template <class SH>
__device__ __forceinline__ int block_excl_scan(int v, SH& sh, int& tot) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  int inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    int n = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += n;
  }
  if (lane == 31) sh.warp_tot[wid] = inc;
  __syncthreads();
  if (wid == 0) {
    int w = sh.warp_tot[lane], winc = w;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      int n = __shfl_up_sync(0xffffffffu, winc, o);
      if (lane >= o) winc += n;
    }
    sh.warp_tot[lane] = winc - w;
    if (lane == 31) sh.total = winc;
  }
  __syncthreads();
  int res = inc - v + sh.warp_tot[wid];
  tot = sh.total;
  __syncthreads();
  return res;
}

// histogram increment with warp aggregation: lanes of a warp that hit the same bin issue ONE atomic (importance
// rows put thousands of elements into a handful of exponent bins; per-element shared-memory atomics on the same
// address serialise).  Called by all 32 lanes; lanes without an element pass take = false.
__device__ __forceinline__ void hist_add_aggregated(uint32_t* hist, bool take, uint32_t bin) {
  const uint32_t key = take ? bin : 0xFFFFFFFFu;
  const uint32_t peers = __match_any_sync(0xffffffffu, key);
  if (take && (int)(threadIdx.x & 31) == __ffs(peers) - 1) atomicAdd(&hist[bin], (uint32_t)__popc(peers));
}

// The K largest values of {val(j) : lo <= j < hi, valid(j)}, ties to the lower index, described as
//   member(j)  <=>  val(j) > thr  ||  (val(j) == thr && j <= cut).
// Requires 0 <= K <= #valid.  All threads of the block call it with uniform arguments.
template <class SH, class F>
__device__ void block_radix_select(F getval, int lo, int hi, int K, SH& sh, uint32_t& thr, int& cut) {
  if (K <= 0) { thr = 0xFFFFFFFFu; cut = -1; return; }
  uint32_t prefix = 0, mask = 0;
  int krem = K;
  int n_eq = 0;
#pragma unroll 1
  for (int pass = 0; pass < 3; ++pass) {
    const int shift = pass == 0 ? 20 : (pass == 1 ? 10 : 0);
    const int nb = pass == 0 ? 4096 : 1024;
    for (int i = threadIdx.x; i < nb; i += ST) sh.hist[i] = 0;
    __syncthreads();
    for (int base = lo; base < hi; base += ST) {  // warp-uniform trip count
      const int j = base + (int)threadIdx.x;
      uint32_t v = 0;
      const bool take = j < hi && getval(j, v) && (v & mask) == prefix;
      hist_add_aggregated(sh.hist, take, (v >> shift) & (uint32_t)(nb - 1));
    }
    __syncthreads();
    // thread t owns w consecutive bins, taken from the top: bins nb-1-t*w-(w-1) .. nb-1-t*w
    const int w = nb / ST;  // 4 or 1
    int cnt[4] = {0, 0, 0, 0}, sum = 0;
    const int top = nb - 1 - (int)threadIdx.x * w;
#pragma unroll
    for (int q = 0; q < 4; ++q)
      if (q < w) { cnt[q] = (int)sh.hist[top - q]; sum += cnt[q]; }
    int tot;
    int excl = block_excl_scan(sum, sh, tot);
    if (excl < krem && krem <= excl + sum) {
      int above = excl;
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        if (q < w) {
          if (above < krem && krem <= above + cnt[q]) { sh.bin = top - q; sh.krem = krem - above; sh.lcut = cnt[q]; }
          above += cnt[q];
        }
      }
    }
    __syncthreads();
    prefix |= (uint32_t)sh.bin << shift;
    mask |= (uint32_t)(nb - 1) << shift;
    krem = sh.krem;
    n_eq = sh.lcut;
    __syncthreads();
  }
  thr = prefix;
  // krem of the n_eq elements equal to thr are taken, lowest indices first
  if (krem >= n_eq) { cut = 0x7FFFFFFF; return; }
  int running = 0;
  int result = -1;
#pragma unroll 1
  for (int base = lo; base < hi; base += ST) {
    const int j = base + (int)threadIdx.x;
    uint32_t v;
    const int flag = (j < hi && getval(j, v) && v == thr) ? 1 : 0;
    int tot;
    const int excl = block_excl_scan(flag, sh, tot);
    if (running + tot >= krem) {
      if (flag && running + excl + 1 == krem) sh.lcut = j;
      __syncthreads();
      result = sh.lcut;
      __syncthreads();
      break;
    }
    running += tot;
  }
  cut = result;
}

__global__ void __launch_bounds__(ST) nacl_select_kernel(const float* __restrict__ imp, const uint32_t* __restrict__ key, int L,
                                                     int k1, int Br, int n_sink, int n_recent, int C,
                                                     int32_t* __restrict__ out_idx) {
  __shared__ SelShared sh;
  const int p = blockIdx.x;
  const uint32_t* ib = reinterpret_cast<const uint32_t*>(imp) + (size_t)p * L;
  const uint32_t* kb = key + (size_t)p * L;
  const int lo = n_sink, hi = L - n_recent;  // non-protected positions [lo, hi)

  // a4: Proxy-Tokens Eviction, top-k1 of the importance outside the protected set
  uint32_t thr_p;
  int cut_p;
  block_radix_select([&](int j, uint32_t& v) { v = ordermap(ib[j]); return true; }, lo, hi, k1, sh, thr_p, cut_p);
  auto in_topk = [&](int j) {
    uint32_t v = ordermap(ib[j]);
    return v > thr_p || (v == thr_p && j <= cut_p);
  };

  // a5: Random Eviction, Gumbel-top-Br over the remaining candidates
  uint32_t thr_r;
  int cut_r;
  block_radix_select([&](int j, uint32_t& v) { if (in_topk(j)) return false; v = kb[j]; return true; },
                     lo, hi, Br, sh, thr_r, cut_r);

  // a6: ascending kept-position list by order-preserving compaction
  int32_t* out = out_idx + (size_t)p * C;
  int running = 0;
#pragma unroll 1
  for (int base = 0; base < L; base += ST) {
    const int j = base + (int)threadIdx.x;
    int keep = 0;
    if (j < L) {
      if (j < lo || j >= hi) keep = 1;
      else if (in_topk(j)) keep = 1;
      else { uint32_t v = kb[j]; keep = (v > thr_r || (v == thr_r && j <= cut_r)) ? 1 : 0; }
    }
    int tot;
    const int excl = block_excl_scan(keep, sh, tot);
    if (keep) {
      const int pos = running + excl;
      if (pos < C) out[pos] = j;
    }
    running += tot;
  }
}

#ifdef NACL_SEL_TRACE
__device__ long long g_sel_trace[16 + 2 * 1024];
__device__ __forceinline__ long long sel_gtimer() { long long t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); return t; }
#define STAMP(k) { if (blockIdx.x == 0 && threadIdx.x == 0) g_sel_trace[k] = clock64(); \
  if (threadIdx.x == 0 && blockIdx.x < 1024 && (k == 0 || k == 5)) g_sel_trace[16 + 2 * blockIdx.x + (k == 5)] = sel_gtimer(); }
#else
#define STAMP(k)
#endif

// ------------------------------------------------------------------ cluster version
// Shared state of one CTA.  Every CTA counts its own slice into a histogram in its own shared memory (warp-
// aggregated).  The cluster then finds the bin that holds the K-th largest value in two small exchanges through
// distributed shared memory instead of merging whole histograms: (1) every CTA pushes the sums of its 64-bin
// super-bins to all ranks; after a cluster barrier every CTA adds them in rank order and finds the super-bin;
// (2) every CTA pushes its 64 bin counts of that super-bin; after a second barrier every CTA finds the bin.
// Integer sums: exact and order-independent.  A buffer is rewritten only after a barrier that every reader reaches
// after its reads, so single buffers suffice.
constexpr int kMaxRanks = 16;
constexpr int kFineW = 68;  // row width of the fine exchange buffer: 64 bins, one neighbour on either side, padding
// strides of K/V and of out_K/out_V in 16-byte vectors; paged source (table != nullptr): row j of batch element b = row
// j % ps of page table[b * tstride + j / ps], page stride sp
struct KvVecLayout { long long sb, sh, sr, ob, oh, orow; const int32_t* table; int ps, tstride; long long sp; };
__device__ __forceinline__ size_t kv_row_vec(const KvVecLayout& ly, int b, int hk, int j) {
  if (ly.table) {
    const long long pg = __ldg(&ly.table[(size_t)b * ly.tstride + j / ly.ps]);
    return (size_t)(pg * ly.sp + hk * ly.sh + (long long)(j % ly.ps) * ly.sr);
  }
  return (size_t)(b * ly.sb + hk * ly.sh + (long long)j * ly.sr);
}
struct ClShared {
  uint32_t hist[HB];
  uint32_t xsup[kMaxRanks][64];   // [rank][super-bin]: pushed by every rank
  uint32_t xfine[kMaxRanks][kFineW];  // [rank][bin of the chosen super-bin] (fast path: one more bin on either side)
  int warp_tot[32];
  int total;
  int sup, bin, krem, neq;        // result of the two steps of a radix pass
  int cnt[3][kMaxRanks];          // per-rank counts: ties of select 0 / select 1, kept positions
  int cut[2];                     // index of the last tie taken, select 0 / select 1
  int lcut;                       // block_radix_select on a candidate list
  int rc[kMaxRanks][4];           // fast path: per-rank counts of the bins threshold-1, threshold, threshold+1
  uint32_t lthr;                  // fast path: threshold value found on a candidate list
  int above;                      // fast path: elements in bins above the threshold bin
  int pad[2];                     // sizeof % 16 == 0
};
static_assert(sizeof(ClShared) % 16 == 0, "the slices behind ClShared stay 16-byte aligned");

// Warp 0: x[r][i], r < nrank, i < n (n = 16 or 64) are per-rank counts of n bins in ascending bin order.  Finds the
// bin that holds the krem-th element counted from the TOP bin; returns (in every lane) its index, the number of
// elements in higher bins and its own count.
template <int W>
__device__ __forceinline__ void warp_find_from_top(const uint32_t (*x)[W], int nrank, int n, int krem, int& idx, int& above,
                                                   int& count) {
  const int lane = threadIdx.x & 31;
  int lo = 0, hi = 0;
  for (int r = 0; r < nrank; ++r) {
    if (lane < n) lo += (int)x[r][lane];
    if (lane + 32 < n) hi += (int)x[r][lane + 32];
  }
  // inclusive suffix sums (bins >= this lane's bin), the high half first
  int shi = hi, slo = lo;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int a = __shfl_down_sync(0xffffffffu, shi, o), b = __shfl_down_sync(0xffffffffu, slo, o);
    if (lane + o < 32) { shi += a; slo += b; }
  }
  const int tot_hi = __shfl_sync(0xffffffffu, shi, 0);
  slo += tot_hi;
  const unsigned mhi = __ballot_sync(0xffffffffu, shi >= krem), mlo = __ballot_sync(0xffffffffu, slo >= krem);
  int l, suf, cnt;
  if (mhi) { l = 31 - __clz(mhi); suf = __shfl_sync(0xffffffffu, shi, l); cnt = __shfl_sync(0xffffffffu, hi, l); idx = 32 + l; }
  else { l = 31 - __clz(mlo); suf = __shfl_sync(0xffffffffu, slo, l); cnt = __shfl_sync(0xffffffffu, lo, l); idx = l; }
  above = suf - cnt;
  count = cnt;
}

// exclusive prefix sum over the block in thread order (ClShared flavour of block_excl_scan)
__device__ __forceinline__ int cl_block_excl_scan(int v, ClShared& sh, int& tot) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  int inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    int n = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += n;
  }
  if (lane == 31) sh.warp_tot[wid] = inc;
  __syncthreads();
  if (wid == 0) {
    int w = sh.warp_tot[lane], winc = w;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      int n = __shfl_up_sync(0xffffffffu, winc, o);
      if (lane >= o) winc += n;
    }
    sh.warp_tot[lane] = winc - w;
    if (lane == 31) sh.total = winc;
  }
  __syncthreads();
  int res = inc - v + sh.warp_tot[wid];
  tot = sh.total;
  __syncthreads();
  return res;
}

// The K largest values of {val(i) : i < nloc on every CTA of the cluster, valid(i)}, ties to the lower global index
// (global index = j0 + i, ascending with the cluster rank), described as
//   member  <=>  val > thr  ||  (val == thr && j <= cut).
// Requires 0 <= K <= #valid.  Every thread of every CTA of the cluster calls it with cluster-uniform K.
// which = 0 / 1 (first / second select).
template <class F>
__device__ void cluster_radix_select(F getval, int nloc, int j0, int K, ClShared& sh, cg::cluster_group& cluster, int which,
                                     uint32_t& thr, int& cut) {
  if (K <= 0) { thr = 0xFFFFFFFFu; cut = -1; return; }
  const unsigned rank = cluster.block_rank(), nrank = cluster.num_blocks();
  const int lane = threadIdx.x & 31;
  uint32_t prefix = 0, mask = 0;
  int krem = K, n_eq = 0;
#pragma unroll 1
  for (int pass = 0; pass < 3; ++pass) {
    const int shift = pass == 0 ? 20 : (pass == 1 ? 10 : 0);
    const int nb = pass == 0 ? 4096 : 1024;
    const int nsup = nb / 64;
#ifdef NACL_SEL_TRACE
#define PSTAMP(k) if (which == 0 && pass == 0 && blockIdx.x == 0 && threadIdx.x == 0) g_sel_trace[8 + k] = clock64();
#else
#define PSTAMP(k)
#endif
    PSTAMP(0)
    for (int i = threadIdx.x; i < nb; i += ST) sh.hist[i] = 0;
    __syncthreads();
    PSTAMP(1)
    for (int base = 0; base < nloc; base += ST) {  // warp-uniform trip count
      const int i = base + (int)threadIdx.x;
      uint32_t v = 0;
      const bool take = i < nloc && getval(i, v) && (v & mask) == prefix;
      if (pass > 0 && !__any_sync(0xffffffffu, take)) continue;  // later digits: most warps hold no element of the bin
      hist_add_aggregated(sh.hist, take, (v >> shift) & (uint32_t)(nb - 1));
    }
    __syncthreads();
    PSTAMP(2)
    // step 1: sums of 64-bin super-bins (thread t: bins 4t..4t+3, 16 lanes per super-bin), pushed to every rank
    {
      int s4 = 0;
      if ((int)threadIdx.x * 4 < nb) {
        const uint4 h = *reinterpret_cast<const uint4*>(&sh.hist[threadIdx.x * 4]);
        s4 = (int)(h.x + h.y + h.z + h.w);
      }
#pragma unroll
      for (int o = 8; o > 0; o >>= 1) s4 += __shfl_xor_sync(0xffffffffu, s4, o);
      const int sb = (int)threadIdx.x >> 4;
      if ((lane & 15) == 0 && sb < nsup)
        for (unsigned r = 0; r < nrank; ++r) cluster.map_shared_rank(&sh, r)->xsup[rank][sb] = (uint32_t)s4;
    }
    PSTAMP(3)
    cluster.sync();
    PSTAMP(4)
    if (threadIdx.x < 32) {
      int idx, above, count;
      warp_find_from_top(sh.xsup, (int)nrank, nsup, krem, idx, above, count);
      if (lane == 0) { sh.sup = idx; sh.krem = krem - above; }
    }
    __syncthreads();
    PSTAMP(5)
    const int sup = sh.sup;
    krem = sh.krem;
    // step 2: the 64 bin counts of that super-bin, pushed to every rank
    if (threadIdx.x < 64) {
      const uint32_t h = sh.hist[sup * 64 + threadIdx.x];
      for (unsigned r = 0; r < nrank; ++r) cluster.map_shared_rank(&sh, r)->xfine[rank][threadIdx.x] = h;
    }
    PSTAMP(6)
    cluster.sync();
    PSTAMP(7)
    if (threadIdx.x < 32) {
      int idx, above, count;
      warp_find_from_top(sh.xfine, (int)nrank, 64, krem, idx, above, count);
      if (lane == 0) { sh.bin = sup * 64 + idx; sh.krem = krem - above; sh.neq = count; }
    }
    __syncthreads();
    prefix |= (uint32_t)sh.bin << shift;
    mask |= (uint32_t)(nb - 1) << shift;
    krem = sh.krem;
    n_eq = sh.neq;
    __syncthreads();
    // every element of the threshold bin is taken: the bin's lower edge is a valid threshold, no need to refine
    if (krem == n_eq) break;  // cluster-uniform
  }
  thr = prefix;
  // krem of the n_eq elements equal to thr are taken, lowest global indices first
  if (krem >= n_eq) { cut = 0x7FFFFFFF; return; }  // cluster-uniform
  int mine = 0;
  for (int i = threadIdx.x; i < nloc; i += ST) {
    uint32_t v;
    mine += (getval(i, v) && v == thr) ? 1 : 0;
  }
  int tot;
  cl_block_excl_scan(mine, sh, tot);
  if (threadIdx.x < nrank) cluster.map_shared_rank(&sh, threadIdx.x)->cnt[which][rank] = tot;
  cluster.sync();
  int before = 0;
  for (unsigned r = 0; r < rank; ++r) before += sh.cnt[which][r];
  const int here = sh.cnt[which][rank];
  if (before < krem && krem <= before + here) {
    // the cut lies in this CTA: the (krem - before)-th tie in index order
    int running = before;
#pragma unroll 1
    for (int base = 0; base < nloc; base += ST) {
      const int i = base + (int)threadIdx.x;
      uint32_t v;
      const int flag = (i < nloc && getval(i, v) && v == thr) ? 1 : 0;
      int t2;
      const int excl = cl_block_excl_scan(flag, sh, t2);
      if (flag && running + excl + 1 == krem)
        for (unsigned r = 0; r < nrank; ++r) cluster.map_shared_rank(&sh, r)->cut[which] = j0 + i;
      running += t2;
      if (running >= krem) break;  // block-uniform
    }
  }
  cluster.sync();
  cut = sh.cut[which];
}


// ------------------------------------------------------------------ fast selection path (one bucket pass per select)
// The general path above refines a 32-bit radix key in three cluster-wide passes per select (two cluster barriers each).
// Here every select takes ONE cluster-wide histogram pass over buckets that are fine where the threshold is expected:
//   top-k:   bucket = the importance's float bits >> 14 (512 buckets per binade) in a 4096-bucket window around the row
//            mean G*P/L (the importance of a head sums to G*P);  the elements of the threshold bucket (a few hundred of
//            32k) are pushed, in index order, into a list that every CTA of the cluster holds, and every CTA finishes the
//            select on that list by itself (no further cluster barrier);
//   sample:  bucket = floor((k~ - lo) * 64) of the fp32 ESTIMATE k~ of the Gumbel key (|k~ - key| < 1e-3, bucket width
//            1/64).  With b the bucket that holds the Br-th largest estimate, the Br-th largest EXACT key lies in
//            [edge(b) - eps, edge(b+1) + eps): every candidate in a bucket >= b+2 is taken, none in a bucket <= b-2 is, and
//            only the candidates of buckets b-1, b, b+1 (some tens) get the exact fp64 key (gumbel_key) and are decided on
//            it -- the same decisions as the general path, bit for bit, at a third of the arithmetic per candidate.
// The path gives up (cluster-uniformly, before it has written anything) whenever a threshold falls into a clamped
// edge bucket or a list would overflow; the general path then runs from the start.
#ifdef NACL_SEL_TRACE
__device__ long long g_sel_trace2[1024][10];
#define FSTAMP(k) { if (blockIdx.x == 0 && threadIdx.x == 0) g_sel_trace[8 + (k)] = clock64(); \
  if (threadIdx.x == 0 && blockIdx.x < 1024) g_sel_trace2[blockIdx.x][k] = sel_gtimer(); }
#else
#define FSTAMP(k)
#endif
__device__ int g_select_fallbacks = 0;  // selections that gave up the fast path (nacl_select_fallbacks)
constexpr int kFastMaxE = 16;   // consecutive positions per thread (instantiations for 8 and 16): slices of at most 16 * ST positions
constexpr int kListCap = 4096;  // candidate-list entries (value, position) per select
// (the top-k bucket drops imp_shift = 12..14 float bits: 512 buckets per binade for rows up to 40k, more for longer rows)
constexpr float kKeyBucketsPerUnit = 64.f, kKeyBelow = 24.f;  // sample buckets: [ln mean - 24, ln mean + 40)

// CODE SIZE matters here: every phase of the selection runs once, so straight-line code is fetched cold (the first
// version of this path spent a third of its time in instruction-fetch stalls).  The helpers are __noinline__ and hand
// their results over in shared memory; loops over ranks and list entries are not unrolled.

// The cluster: the bucket that holds the krem-th element counted from the top bucket of a 4096-bin histogram (sh.hist,
// this CTA's slice), by the two small exchanges of cluster_radix_select; the second one also carries the two bins next
// to the chosen super-bin.  Result in shared memory (valid until the next call): sh.bin, sh.krem = rank inside the bin
// counted from its top, sh.above = elements in higher bins, and for every rank r the counts of bins bin-1, bin, bin+1 of
// ITS slice in sh.rc[r][0..2].
__device__ __noinline__ void fast_hist_find(ClShared& sh, int krem) {
  cg::cluster_group cluster = cg::this_cluster();
  const unsigned rank = cluster.block_rank(), nrank = cluster.num_blocks();
  const int lane = threadIdx.x & 31;
  {
    const uint4 h = *reinterpret_cast<const uint4*>(&sh.hist[threadIdx.x * 4]);
    int s4 = (int)(h.x + h.y + h.z + h.w);
#pragma unroll
    for (int o = 8; o > 0; o >>= 1) s4 += __shfl_xor_sync(0xffffffffu, s4, o);
    const int sb = (int)threadIdx.x >> 4;
    if ((lane & 15) == 0) {
#pragma unroll 1
      for (unsigned r = 0; r < nrank; ++r) cluster.map_shared_rank(&sh, r)->xsup[rank][sb] = (uint32_t)s4;
    }
  }
  cluster.sync();
  if (threadIdx.x < 32) {
    int idx, above, count;
    warp_find_from_top(sh.xsup, (int)nrank, 64, krem, idx, above, count);
    if (lane == 0) { sh.sup = idx; sh.krem = krem - above; sh.above = above; }
  }
  __syncthreads();
  const int sup = sh.sup;
  const int krem1 = sh.krem, above1 = sh.above;
  if (threadIdx.x < 66) {
    const int bq = sup * 64 - 1 + (int)threadIdx.x;  // the 64 bins of the super-bin and one on either side
    const uint32_t h = (bq >= 0 && bq < HB) ? sh.hist[bq] : 0u;
#pragma unroll 1
    for (unsigned r = 0; r < nrank; ++r) cluster.map_shared_rank(&sh, r)->xfine[rank][threadIdx.x] = h;
  }
  cluster.sync();
  if (threadIdx.x < 32) {
    int idx, above, count;
    // (xfine rows are 66 wide here; warp_find_from_top reads columns 1..64 through the shifted base)
    warp_find_from_top(reinterpret_cast<const uint32_t(*)[kFineW]>(&sh.xfine[0][1]), (int)nrank, 64, krem1, idx, above, count);
    if (lane == 0) { sh.bin = sup * 64 + idx; sh.krem = krem1 - above; sh.above = above1 + above; }
    if (lane < (int)nrank) {
      const int q = idx + 1;  // column of the threshold bin
      sh.rc[lane][0] = (int)sh.xfine[lane][q - 1];
      sh.rc[lane][1] = (int)sh.xfine[lane][q];
      sh.rc[lane][2] = (int)sh.xfine[lane][q + 1];
    }
  }
  __syncthreads();
}

// The K-th largest value of list[0..n) (.x = value, ties: the lower list position first), 1 <= K <= n <= kListCap; the
// list is identical in every CTA, every CTA computes the same.  Result in shared memory: sh.lthr = that value, sh.lcut =
// the position of the last tie taken (0x7FFFFFFF: all of them).
__device__ __noinline__ void list_select(const uint2* list, int n, int K, ClShared& sh) {
  if (n <= 256) {
    // rank by counting: the element that exactly K-1 elements precede in (value desc, position asc) order
    if ((int)threadIdx.x < n) {
      const uint32_t me = list[threadIdx.x].x;
      int before = 0;
#pragma unroll 4
      for (int q = 0; q < n; ++q) {
        const uint32_t o = list[q].x;
        before += (o > me || (o == me && q < (int)threadIdx.x)) ? 1 : 0;
      }
      if (before == K - 1) { sh.lthr = me; sh.lcut = (int)threadIdx.x; }
    }
    __syncthreads();
    return;
  }
  uint32_t thr;
  int cutpos;
  block_radix_select([&](int q, uint32_t& v) { v = list[q].x; return true; }, 0, n, K, sh, thr, cutpos);
  if (threadIdx.x == 0) { sh.lthr = thr; sh.lcut = cutpos; }
  __syncthreads();
}

__device__ __noinline__ int fast_scan(int v, ClShared& sh) {
  int tot;
  return block_excl_scan(v, sh, tot);  // (the total stays in sh.total)
}
__device__ __noinline__ float key_estimate_call(float imp, uint32_t j, uint32_t hk, uint32_t b, uint32_t layer, uint32_t k0, uint32_t k1,
                                                uint32_t flags) {
  return gumbel_key_estimate(imp, j, hk, b, layer, k0, k1, flags);
}
// this CTA's entries [off, off + cnt) of the candidate list, already in its own copy, go to the other CTAs' copies
__device__ __noinline__ void list_publish(uint2* list, int off, int cnt) {
  cg::cluster_group cluster = cg::this_cluster();
  const unsigned rank = cluster.block_rank(), nrank = cluster.num_blocks();
  __syncthreads();
#pragma unroll 1
  for (int q = threadIdx.x; q < cnt; q += ST) {
    const uint2 c = list[off + q];
#pragma unroll 1
    for (unsigned r = 0; r < nrank; ++r)
      if (r != rank) cluster.map_shared_rank(list, r)[off + q] = c;
  }
  cluster.sync();
}

// Fast path of the cluster kernel (see above).  Returns false (cluster-uniform) when it gives up; otherwise the kept
// positions are in out[] and ib[0..tot) (this CTA's part, output rows base .. base+tot).
template <int FE>
__device__ bool select_fast(const float* __restrict__ row, int nloc, int E, int j0, int lo, int hi, int k1, int Br, int C,
                            int imp_base, int imp_shift, float key_lo, uint32_t hk_g, uint32_t b_g, uint32_t layer, uint32_t sk0, uint32_t sk1,
                            uint32_t flags, ClShared& sh, uint32_t* ib, uint32_t* kb, uint2* list, cg::cluster_group& cluster,
                            int32_t* __restrict__ out, int& tot_out, int& base_out) {
  const unsigned rank = cluster.block_rank(), nrank = cluster.num_blocks();
  // thread t owns the E = ceil(Lc / ST) <= FE consecutive positions from i0 = t * E on (short slices spread over all threads)
  const int t = (int)threadIdx.x, i0 = t * E;
  auto free_pos = [&](int i) { const int j = j0 + i; return j >= lo && j < hi; };

  // coalesced load through shared memory, then the thread's consecutive positions in registers
  for (int i = t; i < nloc; i += ST) ib[i] = ordermap(__float_as_uint(row[i]));
  __syncthreads();
  uint32_t v[FE];
  uint32_t livem = 0, freem = 0;  // bit e: position i0+e is this thread's and exists / and is not protected
#pragma unroll
  for (int e = 0; e < FE; ++e) {
    const bool live = e < E && i0 + e < nloc;
    v[e] = live ? ib[i0 + e] : 0u;
    livem |= (live ? 1u : 0u) << e;
    freem |= (live && free_pos(i0 + e) ? 1u : 0u) << e;
  }
  STAMP(1)

  // ---- a4: top-k1 of the importance outside the protected set
  uint32_t thr_p = 0xFFFFFFFFu;
  int cut_p = -1;
  uint32_t inb = 0;  // bit e: in the threshold bucket (after the find)
  int dg[FE];
  if (k1 > 0) {
    for (int i = t; i < HB; i += ST) sh.hist[i] = 0;
    __syncthreads();
#pragma unroll
    for (int e = 0; e < FE; ++e) {
      dg[e] = min(max((int)(v[e] >> imp_shift) - imp_base, 0), HB - 1);
      // (plain shared-memory atomics: the buckets are fine where the values are, lanes rarely meet in one)
      if ((freem >> e) & 1u) atomicAdd(&sh.hist[dg[e]], 1u);
    }
    __syncthreads();
    FSTAMP(0)
  }
  // every CTA of the cluster is running (the barrier it arrived at when it started): its shared memory may be written
#ifndef NACL_SEL_NO_SPLIT_BARRIER
  asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
#else
  cluster.sync();
#endif
  if (k1 > 0) {
    fast_hist_find(sh, k1);
    FSTAMP(1)
    const int bin = sh.bin, krem = sh.krem;
    int n_eq = 0, before = 0;
#pragma unroll 1
    for (unsigned r = 0; r < nrank; ++r) { before += r < rank ? sh.rc[r][1] : 0; n_eq += sh.rc[r][1]; }
    if (bin == 0 || bin == HB - 1 || n_eq > kListCap) return false;  // clamped bucket / list overflow (cluster-uniform)
    if (krem == n_eq) {
      thr_p = (uint32_t)(bin + imp_base) << imp_shift;  // the whole bucket is taken: its lower edge is a threshold
      cut_p = 0x7FFFFFFF;
    } else {
      int mine = 0;
#pragma unroll
      for (int e = 0; e < FE; ++e) {
        const bool b = ((freem >> e) & 1u) && dg[e] == bin;
        inb |= (b ? 1u : 0u) << e;
        mine += b ? 1 : 0;
      }
      int pos = before + fast_scan(mine, sh);
#pragma unroll
      for (int e = 0; e < FE; ++e)
        if ((inb >> e) & 1u) list[pos++] = make_uint2(v[e], (uint32_t)(j0 + i0 + e));
      list_publish(list, before, (int)sh.rc[rank][1]);
      FSTAMP(2)
      list_select(list, n_eq, krem, sh);
      thr_p = sh.lthr;
      cut_p = sh.lcut == 0x7FFFFFFF ? 0x7FFFFFFF : (int)list[sh.lcut].y;
      FSTAMP(3)
    }
  }
  auto in_topk = [&](uint32_t val, int j) { return val > thr_p || (val == thr_p && j <= cut_p); };
  STAMP(2)
  // ---- a5: Gumbel-top-Br over the remaining candidates
  int kbin = -1;                 // bucket of the Br-th largest key estimate
  uint32_t thr_r = 0xFFFFFFFFu;  // exact threshold among the candidates of buckets kbin-1 .. kbin+1
  int cut_r = -1;
  int kd[FE];                    // bucket of the key estimate; -1: not a candidate
#pragma unroll
  for (int e = 0; e < FE; ++e) kd[e] = -1;
  if (Br > 0) {
    // (no barrier needed here: a CTA writes another CTA's exchange buffers or list again only after the cluster barriers of
    // the next fast_hist_find, which that CTA reaches after its last read of them)
    for (int i = t; i < HB; i += ST) sh.hist[i] = 0;
    __syncthreads();
#pragma unroll
    for (int e = 0; e < FE; ++e) {
      const int i = i0 + e;
      if (((freem >> e) & 1u) && !in_topk(v[e], j0 + i)) {
        const float w = __uint_as_float(v[e] & 0x80000000u ? v[e] & 0x7FFFFFFFu : ~v[e]);  // ordermap^-1
        const float ke = key_estimate_call(w, (uint32_t)(j0 + i), hk_g, b_g, layer, sk0, sk1, flags);
        // (-inf, and anything below the window, lands in bucket 0; NaN cannot occur: the weight is >= 0 or +inf)
        kd[e] = (int)fminf(fmaxf((ke - key_lo) * kKeyBucketsPerUnit, 0.f), (float)(HB - 1));
        atomicAdd(&sh.hist[kd[e]], 1u);
      }
    }
    STAMP(3)
    __syncthreads();
    FSTAMP(4)
    fast_hist_find(sh, Br);
    FSTAMP(5)
    kbin = sh.bin;
    const int above = sh.above;
    int n_mid = 0, n_up = 0, before = 0;
#pragma unroll 1
    for (unsigned r = 0; r < nrank; ++r) {
      const int c3 = sh.rc[r][0] + sh.rc[r][1] + sh.rc[r][2];
      before += r < rank ? c3 : 0;
      n_mid += c3;
      n_up += sh.rc[r][2];
    }
    if (kbin < 2 || kbin > HB - 3 || n_mid > kListCap) return false;  // too close to a clamped bucket / list overflow
    const int m = Br - (above - n_up);  // to be taken from buckets kbin-1 .. kbin+1: all of the buckets >= kbin+2 are in
    uint32_t midm = 0;
    int mine = 0;
#pragma unroll
    for (int e = 0; e < FE; ++e) {
      const bool b = kd[e] >= kbin - 1 && kd[e] <= kbin + 1;
      midm |= (b ? 1u : 0u) << e;
      mine += b ? 1 : 0;
    }
    // the candidates of the three buckets go out as (importance, position); every CTA then evaluates the exact keys of the
    // WHOLE list, one per thread in converged warps (a few tens of keys: cheaper than each owner evaluating its own in
    // divergent code), and the owners read theirs back from their list slot
    const int pos0 = before + fast_scan(mine, sh);
    {
      int pos = pos0;
#pragma unroll
      for (int e = 0; e < FE; ++e)
        if ((midm >> e) & 1u) list[pos++] = make_uint2(v[e], (uint32_t)(j0 + i0 + e));
    }
    list_publish(list, before, sh.rc[rank][0] + sh.rc[rank][1] + sh.rc[rank][2]);
    FSTAMP(6)
#pragma unroll 1
    for (int q = t; q < n_mid; q += ST) {
      const uint2 c = list[q];
      const float w = __uint_as_float(c.x & 0x80000000u ? c.x & 0x7FFFFFFFu : ~c.x);  // ordermap^-1
      list[q].x = gumbel_key<true>(w, c.y, hk_g, b_g, layer, sk0, sk1, flags);       // exact, order-mapped
    }
    __syncthreads();
    FSTAMP(7)
    list_select(list, n_mid, m, sh);
    thr_r = sh.lthr;
    cut_r = sh.lcut == 0x7FFFFFFF ? 0x7FFFFFFF : (int)list[sh.lcut].y;
    // the owners decide their candidates of the three buckets on the exact key in their list slot
    {
      int q = pos0;
#pragma unroll
      for (int e = 0; e < FE; ++e)
        if ((midm >> e) & 1u) {
          const uint32_t kx = list[q++].x;
          kd[e] = (kx > thr_r || (kx == thr_r && j0 + i0 + e <= cut_r)) ? HB : -1;  // HB: "above the threshold"
        }
    }
  }

  STAMP(4)
  // ---- a6: ascending kept-position list
  uint32_t keep = 0;
  int mine = 0;
#pragma unroll
  for (int e = 0; e < FE; ++e) {
    const int i = i0 + e;
    bool k = false;
    if ((livem >> e) & 1u) k = !((freem >> e) & 1u) || in_topk(v[e], j0 + i) || kd[e] >= kbin + 2;
    keep |= (k ? 1u : 0u) << e;
    mine += k ? 1 : 0;
  }
  const int excl = fast_scan(mine, sh);
  const int tot = sh.total;
  __syncthreads();  // (ib is rewritten below; its last reads lie before the scan)
  if (t < (int)nrank) cluster.map_shared_rank(&sh, t)->cnt[2][rank] = tot;
  FSTAMP(8)
  cluster.sync();  // the last access to another CTA's shared memory lies before this barrier
  FSTAMP(9)
  int base = 0;
#pragma unroll 1
  for (unsigned r = 0; r < rank; ++r) base += sh.cnt[2][r];
  int pos = base + excl;
#pragma unroll
  for (int e = 0; e < FE; ++e)
    if ((keep >> e) & 1u) {
      if (pos < C) { out[pos] = j0 + i0 + e; ib[pos - base] = (uint32_t)(j0 + i0 + e); }
      ++pos;
    }
  tot_out = tot;
  base_out = base;
  return true;
}

// One cluster per (batch, kv head); CTA `rank` owns positions [rank*Lc, min(L, (rank+1)*Lc)).
// Dynamic shared memory: ClShared, uint32 ib[Lc] (order-mapped importance), uint32 kb[Lc] (order-mapped keys, later keep flags).
__global__ void __launch_bounds__(ST) nacl_select_cluster_kernel(const float* __restrict__ imp, int Hkv, int L, int Lc, int k1, int Br,
                                                                 int n_sink, int n_recent, int C, uint32_t sk0, uint32_t sk1,
                                                                 uint32_t layer, uint32_t flags, int32_t* __restrict__ out_idx,
                                                                 const int4* Kv, const int4* Vv, int4* oKv, int4* oVv, int vpr,
                                                                 uint32_t b_off, uint32_t h_off, KvVecLayout ly, int fast,
                                                                 int imp_base, int imp_shift, float key_lo, int inplace) {
  cg::cluster_group cluster = cg::this_cluster();
  extern __shared__ __align__(16) unsigned char dyn_raw[];
  ClShared& sh = *reinterpret_cast<ClShared*>(dyn_raw);
  uint32_t* dyn = reinterpret_cast<uint32_t*>(dyn_raw + sizeof(ClShared));
  const unsigned rank = cluster.block_rank(), nrank = cluster.num_blocks();
  const int p = blockIdx.x / nrank;  // b * Hkv + hk
  const int b = p / Hkv, hk = p - b * Hkv;
  const int j0 = (int)rank * Lc;
  const int nloc = max(0, min(L - j0, Lc));
  uint32_t* ib = dyn;
  uint32_t* kb = dyn + Lc;
  const int lo = n_sink, hi = L - n_recent;  // non-protected positions [lo, hi)
  const float* row = imp + (size_t)p * L + j0;

  int tot = 0, base = 0;
  int32_t* out = out_idx + (size_t)p * C;
  STAMP(0)
  bool done = false;
  if (fast) {
    // split cluster barrier: arrive now, wait right before the first write into another CTA's shared memory (select_fast)
#ifndef NACL_SEL_NO_SPLIT_BARRIER
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
#endif
    uint2* list = reinterpret_cast<uint2*>(dyn + 2 * (size_t)Lc);
    const int E = (Lc + ST - 1) / ST;
    if (E <= 8)
      done = select_fast<8>(row, nloc, E, j0, lo, hi, k1, Br, C, imp_base, imp_shift, key_lo, (uint32_t)hk + h_off, (uint32_t)b + b_off, layer, sk0,
                            sk1, flags, sh, ib, kb, list, cluster, out, tot, base);
    else
      done = select_fast<16>(row, nloc, E, j0, lo, hi, k1, Br, C, imp_base, imp_shift, key_lo, (uint32_t)hk + h_off, (uint32_t)b + b_off, layer, sk0,
                             sk1, flags, sh, ib, kb, list, cluster, out, tot, base);
  }
  if (!done) {
  if (fast && rank == 0 && threadIdx.x == 0) atomicAdd(&g_select_fallbacks, 1);
  for (int i = threadIdx.x; i < nloc; i += ST) ib[i] = ordermap(__float_as_uint(row[i]));
  cluster.sync();  // every CTA of the cluster is running: its shared memory may be written
  STAMP(1)
  auto free_pos = [&](int i) { const int j = j0 + i; return j >= lo && j < hi; };

  // a4: Proxy-Tokens Eviction, top-k1 of the importance outside the protected set
  uint32_t thr_p;
  int cut_p;
  cluster_radix_select([&](int i, uint32_t& v) { v = ib[i]; return free_pos(i); }, nloc, j0, k1, sh, cluster, 0, thr_p, cut_p);
  auto in_topk = [&](int i) {
    const uint32_t v = ib[i];
    return v > thr_p || (v == thr_p && j0 + i <= cut_p);
  };
  STAMP(2)

  // a5: Random Eviction, Gumbel-top-Br over the remaining candidates; keys only for those
  if (Br > 0) {
    // four independent fp64 log chains per thread in flight
    for (int base = 0; base < nloc; base += 4 * ST) {
      uint32_t kk[4];
      bool cand[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int i = base + u * ST + (int)threadIdx.x;
        cand[u] = i < nloc && free_pos(i) && !in_topk(i);
        if (cand[u])
          kk[u] = gumbel_key(row[i], (uint32_t)(j0 + i), (uint32_t)hk + h_off, (uint32_t)b + b_off, layer, sk0, sk1, flags);
      }
#pragma unroll
      for (int u = 0; u < 4; ++u)
        if (cand[u]) kb[base + u * ST + (int)threadIdx.x] = kk[u];
    }
    __syncthreads();
  }
  STAMP(3)
  uint32_t thr_r;
  int cut_r;
  cluster_radix_select([&](int i, uint32_t& v) { if (!free_pos(i) || in_topk(i)) return false; v = kb[i]; return true; },
                       nloc, j0, Br, sh, cluster, 1, thr_r, cut_r);

  STAMP(4)
  // a6: ascending kept-position list: keep flags, then ONE block scan over threads that own consecutive positions,
  // exclusive offsets over the cluster ranks, compaction
  for (int i = threadIdx.x; i < nloc; i += ST) {
    int keep;
    if (!free_pos(i) || in_topk(i)) keep = 1;
    else { const uint32_t v = kb[i]; keep = (v > thr_r || (v == thr_r && j0 + i <= cut_r)) ? 1 : 0; }
    kb[i] = (uint32_t)keep;
  }
  __syncthreads();
  const int E = (Lc + ST - 1) / ST;  // consecutive positions per thread
  const int i0 = (int)threadIdx.x * E;
  int mine = 0;
  for (int e = 0; e < E; ++e) mine += (i0 + e < nloc) ? (int)kb[i0 + e] : 0;
  const int excl = cl_block_excl_scan(mine, sh, tot);
  if (threadIdx.x < nrank) cluster.map_shared_rank(&sh, threadIdx.x)->cnt[2][rank] = tot;
  cluster.sync();  // the last access to another CTA's shared memory lies before this barrier
  for (unsigned r = 0; r < rank; ++r) base += sh.cnt[2][r];  // kept positions of the lower ranks
  int pos = base + excl;
  for (int e = 0; e < E; ++e) {
    const int i = i0 + e;
    if (i < nloc && kb[i]) {
      if (pos < C) { out[pos] = j0 + i; ib[pos - base] = (uint32_t)(j0 + i); }  // (ib is free: the keep flags are final)
      ++pos;
    }
  }
  }  // general path
  STAMP(5)
  if (vpr == 0) return;
  // a7, fused: this CTA moves the K and V rows of the positions IT kept (out rows base .. base+tot), 16-byte vectors,
  // consecutive threads on consecutive vectors of the output, four vectors of K and of V in flight per thread
  __syncthreads();
  const int n_vec = min(tot, C - base) * vpr;
  // K/V and the outputs have their own strides (in 16-byte vectors); a row's vpr vectors are contiguous
  const size_t dst0 = (size_t)(b * ly.ob + hk * ly.oh + (long long)base * ly.orow);
  const long long dpad = ly.orow - vpr;  // 0 for contiguous output rows: then the output vector index is just v
  if (dpad == 0) {
    int start_vec = 0;
    if (inplace) {
      // In-place compaction (out_K == K, out_V == V, same strides): output row c receives position S[c] >= c, so a write
      // can only destroy a row that is the SOURCE of an output row at or before it.  The rows whose source lies below C
      // (a prefix of every CTA's ascending list) are moved first, in ascending order: rank after rank, chunk after chunk,
      // all loads of a chunk before its stores.  Every other row has its source at or above C, where nothing is written:
      // those move in parallel afterwards.
      int nr = 0;
      {
        int lo_ = 0, hi_ = n_vec / vpr;
        while (lo_ < hi_) {
          const int mid = (lo_ + hi_) >> 1;
          if ((int)ib[mid] < C) lo_ = mid + 1; else hi_ = mid;
        }
        nr = lo_;
      }
      const int risk_vec = nr * vpr;
      for (unsigned r = 0; r < nrank; ++r) {
        if (rank == r) {
          for (int c0 = 0; c0 < risk_vec; c0 += ST * 4) {  // block-uniform trip count
            size_t src[4];
            int4 a[4], b4[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
              const int v = c0 + (int)threadIdx.x + u * ST;
              if (v < risk_vec) {
                const int row = v / vpr;
                src[u] = kv_row_vec(ly, b, hk, (int)ib[row]) + (v - row * vpr);
                a[u] = __ldcs(Kv + src[u]);
                b4[u] = __ldcs(Vv + src[u]);
              }
            }
            __syncthreads();
#pragma unroll
            for (int u = 0; u < 4; ++u) {
              const int v = c0 + (int)threadIdx.x + u * ST;
              if (v < risk_vec) { __stcs(oKv + dst0 + v, a[u]); __stcs(oVv + dst0 + v, b4[u]); }
            }
            __syncthreads();
          }
        }
        cluster.sync();
      }
      start_vec = risk_vec;
    }
    // four vectors of K and four of V in flight per thread
    for (int v0 = start_vec + threadIdx.x; v0 < n_vec; v0 += ST * 4) {
      size_t src[4];
      int4 a[4], b4[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int v = v0 + u * ST;
        if (v < n_vec) {
          const int row = v / vpr;
          src[u] = kv_row_vec(ly, b, hk, (int)ib[row]) + (v - row * vpr);
        }
      }
#pragma unroll
      for (int u = 0; u < 4; ++u)
        if (v0 + u * ST < n_vec) { a[u] = __ldcs(Kv + src[u]); b4[u] = __ldcs(Vv + src[u]); }
#pragma unroll
      for (int u = 0; u < 4; ++u)
        if (v0 + u * ST < n_vec) { __stcs(oKv + dst0 + v0 + u * ST, a[u]); __stcs(oVv + dst0 + v0 + u * ST, b4[u]); }
    }
    return;
  }
  // output rows with a stride of their own (a cache with spare capacity, a token-major destination): K, then V
  for (int v0 = threadIdx.x; v0 < n_vec; v0 += ST * 4) {
    size_t src[4], dst[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int v = v0 + u * ST;
      if (v < n_vec) {
        const int row = v / vpr;
        src[u] = kv_row_vec(ly, b, hk, (int)ib[row]) + (v - row * vpr);
        dst[u] = dst0 + (size_t)v + (size_t)(row * dpad);
      }
    }
#pragma unroll
    for (int t = 0; t < 2; ++t) {
      const int4* __restrict__ in = t ? Vv : Kv;
      int4* __restrict__ out = t ? oVv : oKv;
      int4 a[4];
#pragma unroll
      for (int u = 0; u < 4; ++u)
        if (v0 + u * ST < n_vec) a[u] = __ldcs(in + src[u]);
#pragma unroll
      for (int u = 0; u < 4; ++u)
        if (v0 + u * ST < n_vec) __stcs(out + dst[u], a[u]);
    }
  }
}

}  // namespace

cudaError_t launch_keys(const float* imp, uint32_t* key, int batch, int Hkv, int L, uint64_t seed, int layer,
                        uint32_t flags, bool ordermapped, int batch_offset, int head_offset, cudaStream_t st) {
  dim3 grid((L + 255) / 256, batch * Hkv);
  const uint32_t sk0 = (uint32_t)(seed & 0xFFFFFFFFu), sk1 = (uint32_t)(seed >> 32);
  if (ordermapped)
    nacl_keys_kernel<true><<<grid, 256, 0, st>>>(imp, key, Hkv, L, sk0, sk1, (uint32_t)layer, flags, (uint32_t)batch_offset, (uint32_t)head_offset);
  else
    nacl_keys_kernel<false><<<grid, 256, 0, st>>>(imp, key, Hkv, L, sk0, sk1, (uint32_t)layer, flags, (uint32_t)batch_offset, (uint32_t)head_offset);
  return cudaGetLastError();
}

// slices of at most this many positions per CTA stay in shared memory (2 x 4 bytes each)
constexpr int kMaxSlice = 20480;

// what the latest launch_select on this host thread decided (nacl_last_select_launch)
static thread_local int g_last_sel_grid = 0, g_last_sel_cluster = 0, g_last_sel_fused = 0;

bool select_uses_cluster(int L) { return (L + kMaxRanks - 1) / kMaxRanks <= kMaxSlice; }

cudaError_t launch_select(const float* imp, uint32_t* key, int batch, int Hkv, int L, int budget_proxy, int budget_random,
                          int n_sink, int n_recent, uint64_t seed, int layer, uint32_t flags, int32_t* out_idx,
                          const void* K, const void* V, void* out_K, void* out_V, int row_bytes, bool* gathered,
                          int batch_offset, int head_offset, const Shape* layout, float imp_mean, bool inplace, cudaStream_t st) {
  *gathered = false;
  const int C = budget_proxy + budget_random;
  if (C == 0) return cudaSuccess;
  const int k1 = budget_proxy - n_sink - n_recent;
  const uint32_t sk0 = (uint32_t)(seed & 0xFFFFFFFFu), sk1 = (uint32_t)(seed >> 32);
  // very long rows, or no cluster size that this device can co-schedule: sampling keys in a kernel of their own, one CTA
  // per head working out of global memory (the caller then runs the stand-alone gather)
  auto long_row_path = [&]() -> cudaError_t {
    g_last_sel_grid = batch * Hkv; g_last_sel_cluster = 0; g_last_sel_fused = 0;
    if (budget_random > 0) {
      StageScope sc(ST_KEYS, st);
      cudaError_t e = launch_keys(imp, key, batch, Hkv, L, seed, layer, flags, true, batch_offset, head_offset, st);
      if (e != cudaSuccess) return e;
    }
    StageScope sc(ST_SELECT, st);
    nacl_select_kernel<<<batch * Hkv, ST, 0, st>>>(imp, key, L, k1, budget_random, n_sink, n_recent, C, out_idx);
    return cudaGetLastError();
  };
  if (!select_uses_cluster(L)) return inplace ? cudaErrorNotSupported : long_row_path();  // in place: the fused gather only
  // cluster size n: the n that minimises (waves of co-resident clusters) x (per-CTA cost ~ fixed + per-position),
  // with the co-residency limit asked from the runtime (clusters need n free SMs inside one GPC)
  cudaLaunchConfig_t cfg = {};
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  cfg.blockDim = dim3(ST);
  cfg.stream = st;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  const long heads = (long)batch * Hkv;
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) { cudaGetLastError(); dev = 0; }
  int n = 0, Lc = 0;
  size_t dyn = 0;
  double best = 0.0;
  // the fast path (slices of at most kFastMaxE * ST positions) keeps a candidate list behind the two slice arrays
  auto dyn_bytes = [](int lc) {
    return sizeof(ClShared) + (size_t)lc * 2 * sizeof(uint32_t) + (lc <= kFastMaxE * ST ? (size_t)kListCap * sizeof(uint2) : 0);
  };
  cudaError_t e = cudaFuncSetAttribute(nacl_select_cluster_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       (int)(sizeof(ClShared) + (size_t)kMaxSlice * 2 * sizeof(uint32_t)));
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(nacl_select_cluster_kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);  // clusters of 16
  if (e != cudaSuccess) return e;
  for (int c = 1; c <= kMaxRanks; c *= 2) {
    const int lc = ((L + c - 1) / c + 3) / 4 * 4;
    if (lc > kMaxSlice) continue;
#ifdef NACL_FORCE_CLUSTER  // diagnostics: one cluster size only
    if (c != NACL_FORCE_CLUSTER) continue;
#endif
    if (c > 1 && L / c < ST / 2) break;  // slices below half a block of positions are not worth a barrier per pass
    // beside other work (nacl_evict_batch): the grid stays below ~45 % of the SMs, so that the other stream's scoring CTAs
    // find room while this selection waits on its barriers (cfg 3 93.1 -> 85.7 us per call, cfg 4 205.6 -> 203.6)
#ifndef NACL_DIAG_NO_SHARE
    if ((flags & NACL_FLAG_SELECT_SHARE_SMS) && n != 0 && heads * c * 20 > (long)kNumSMs * 9) break;
#endif
    const size_t d = dyn_bytes(lc);
    // co-resident clusters of this size, per device and shared-memory class; -1: the device cannot schedule one (a MIG
    // slice, another SKU): the size is skipped
    static std::mutex cache_mu;
    static int active_cache[64][5][2] = {};
    const int ci = c == 1 ? 0 : (c == 2 ? 1 : (c == 4 ? 2 : (c == 8 ? 3 : 4))), si = d > 100 * 1024 ? 1 : 0;
    int active;
    {
      std::lock_guard<std::mutex> lk(cache_mu);
      active = active_cache[dev][ci][si];
      if (active == 0) {
        cfg.gridDim = dim3((unsigned)(c * 64));
        cfg.dynamicSmemBytes = si ? sizeof(ClShared) + (size_t)kMaxSlice * 2 * sizeof(uint32_t) : 100 * 1024;
        attr[0].val.clusterDim.x = (unsigned)c;
        if (cudaOccupancyMaxActiveClusters(&active, nacl_select_cluster_kernel, &cfg) != cudaSuccess || active < 1) {
          cudaGetLastError();
          active = -1;
        }
        active_cache[dev][ci][si] = active;
      }
    }
    if (active < 1) continue;
    const double waves = (double)((heads + active - 1) / active);
    // cycles per wave, measured at cfg 4 (profiles/): the one-pass bucket path where the slice allows it, else the general one
    const bool fast_ok = lc <= kFastMaxE * ST && !(flags & NACL_FLAG_SELECT_GENERAL);
    const double cost = waves * (fast_ok ? 20000.0 + 4.0 * lc : 37000.0 + 6.0 * lc);
    if (n == 0 || cost < best) { n = c; Lc = lc; dyn = d; best = cost; }
  }
  if (n == 0) return inplace ? cudaErrorNotSupported : long_row_path();
  cfg.gridDim = dim3((unsigned)(heads * n));
  cfg.dynamicSmemBytes = dyn;
  attr[0].val.clusterDim.x = (unsigned)n;
  KvVecLayout ly{};
  if (K != nullptr) {
    const long long epv = 16 / layout->esize;
    ly = KvVecLayout{layout->kv_sb / epv, layout->kv_sh / epv, layout->kv_sr / epv, layout->o_sb / epv, layout->o_sh / epv, layout->o_sr / epv,
                     layout->table, layout->ps, layout->tstride, layout->kv_sp / epv};
  }
  // fast path: bucket windows around the row mean of the importance (its sum over a row is known: G*P) and around the
  // logarithm of that mean for the sampling keys (uniform weights: ln w = 0; weight exp(imp): ln w = imp)
  int fast = (Lc <= kFastMaxE * ST && !(flags & NACL_FLAG_SELECT_GENERAL) && imp_mean > 0.f && imp_mean < 1e30f) ? 1 : 0;
  int imp_base = 0, imp_shift = 14;
  float key_lo = 0.f;
  if (fast) {
    uint32_t mb;
    memcpy(&mb, &imp_mean, sizeof(mb));
    // finer buckets for longer rows (the threshold bucket should hold a few hundred elements at most); the window is
    // centred on the mean: a skewed row (few heavy hitters carry the mass) has its top-k threshold well BELOW the mean
    imp_shift = L <= 40000 ? 14 : (L <= 80000 ? 13 : 12);
    imp_base = (int)((mb | 0x80000000u) >> imp_shift) - HB / 2;
    const float centre = (flags & NACL_FLAG_SAMPLE_UNIFORM) ? 0.f : ((flags & NACL_FLAG_SAMPLE_SOFTMAX_OF_SCORE) ? imp_mean : logf(imp_mean));
    key_lo = centre - kKeyBelow;
  }
  // the kernel also moves the kept rows when its grid covers most of the GPU; a grid of few CTAs (few heads, short rows)
  // would leave the gather to a fraction of the SMs: the stand-alone gather kernel (all SMs) follows instead
  // ... except beside other work (nacl_evict_batch) when the scoring is short and HBM-bound (G*P <= 128): there the small grid
  // that keeps its SMs for the gather beats a second kernel that competes with the other stream's sweeps for all SMs
  // (cfg 2 42.7 -> 39.9 us per call, cfg 3 86.5 -> 84.5; at G*P = 256: cfg 4 +0.5, cfg 5 +10)
  const bool small_grid_fused = (flags & NACL_FLAG_SELECT_SHARE_SMS) && layout != nullptr && layout->rows <= 128;
#ifdef NACL_DIAG_FUSE_GATHER  // diagnostics: the fused gather whatever the grid size
  *gathered = K != nullptr && (inplace || !(flags & NACL_FLAG_GATHER_SEPARATE));
#else
  *gathered = K != nullptr && (inplace || (!(flags & NACL_FLAG_GATHER_SEPARATE) && (heads * n * 5 >= (long)kNumSMs * 4 || small_grid_fused)));
#endif
  g_last_sel_grid = (int)(heads * n); g_last_sel_cluster = n; g_last_sel_fused = *gathered ? 1 : 0;
  {
    StageScope sc(ST_SELECT, st);
    e = cudaLaunchKernelEx(&cfg, nacl_select_cluster_kernel, imp, Hkv, L, Lc, k1, budget_random, n_sink, n_recent, C, sk0, sk1,
                           (uint32_t)layer, flags, out_idx, (const int4*)K, (const int4*)V, (int4*)out_K, (int4*)out_V,
                           *gathered ? row_bytes / 16 : 0, (uint32_t)batch_offset, (uint32_t)head_offset, ly, fast, imp_base, imp_shift, key_lo,
                           inplace ? 1 : 0);
  }
  if (e == cudaSuccess || inplace) return e;
  // the launch itself was refused (cluster resources): nothing ran; take the path without clusters
  cudaGetLastError();
  *gathered = false;
  return long_row_path();
}

// 4-byte words of the `key` scratch the select needs (long-row path: the keys)
size_t select_scratch_words(int batch, int Hkv, int L) {
  // the keys of the path without clusters (very long rows, or a device that cannot co-schedule a cluster); the cluster
  // path keeps everything in shared memory
  return (size_t)batch * Hkv * L + 64;
}

}  // namespace nacl

extern "C" __attribute__((visibility("default"))) void nacl_last_select_launch(int* grid_ctas, int* cluster_size, int* fused_gather) {
  if (grid_ctas) *grid_ctas = nacl::g_last_sel_grid;
  if (cluster_size) *cluster_size = nacl::g_last_sel_cluster;
  if (fused_gather) *fused_gather = nacl::g_last_sel_fused;
}

extern "C" __attribute__((visibility("default"))) int nacl_select_fallbacks(int reset) {
  int v = 0;
  if (cudaMemcpyFromSymbol(&v, nacl::g_select_fallbacks, sizeof(v)) != cudaSuccess) { cudaGetLastError(); return NACL_ERR_CUDA; }
  if (reset) {
    const int zero = 0;
    if (cudaMemcpyToSymbol(nacl::g_select_fallbacks, &zero, sizeof(zero)) != cudaSuccess) { cudaGetLastError(); return NACL_ERR_CUDA; }
  }
  return v;
}

#ifdef NACL_SEL_TRACE
extern "C" __attribute__((visibility("default"))) int nacl_debug_sel_trace_reset() {
  static long long zeros[16 + 2 * 1024] = {};
  return (int)cudaMemcpyToSymbol(nacl::g_sel_trace, zeros, sizeof(zeros));
}
extern "C" __attribute__((visibility("default"))) int nacl_debug_sel_trace2_read(long long* host) {
  return (int)cudaMemcpyFromSymbol(host, nacl::g_sel_trace2, sizeof(nacl::g_sel_trace2));
}
extern "C" __attribute__((visibility("default"))) int nacl_debug_sel_trace_read(long long* host) {
  return (int)cudaMemcpyFromSymbol(host, nacl::g_sel_trace, sizeof(nacl::g_sel_trace));
}
#endif
