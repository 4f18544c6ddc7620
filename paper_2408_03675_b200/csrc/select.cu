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
//   nacl_select_cluster_kernel: the same selection with one thread-block CLUSTER (1..8 CTAs) per (batch, kv head):
//                  every CTA keeps its slice of the importance row and of the sampling keys in shared memory,
//                  the radix histograms of the slices meet in the shared memory of the cluster's rank-0 CTA
//                  (distributed shared memory), and the keys are computed in the same kernel, only for the
//                  candidates that survive the top-k.  Used whenever the slices fit; 8x more CTAs than heads.
// Integer work only after the keys: results are bit-exact functions of (imp, key).
#include <cooperative_groups.h>

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
    uint32_t hi0 = __umulhi(M0, c0), lo0 = M0 * c0;
    uint32_t hi1 = __umulhi(M1, c2), lo1 = M1 * c2;
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

// order-mapped Gumbel-top-k key of position j of kv head hk of batch element b (R4/R5/R10/R13/R15)
__device__ __forceinline__ uint32_t gumbel_key(float imp, uint32_t j, uint32_t hk, uint32_t b, uint32_t layer, uint32_t k0, uint32_t k1,
                                               uint32_t flags) {
  const uint32_t x = philox4x32_10_word0(j, hk, b, layer, k0, k1);
  const double u = ((double)(x >> 9) + 0.5) * 0x1p-23;  // exact; u in [2^-24, 1-2^-24]
  const double w = (double)imp;
  double ln_w;
  if (flags & NACL_FLAG_SAMPLE_UNIFORM) ln_w = 0.0;
  else if (flags & NACL_FLAG_SAMPLE_SOFTMAX_OF_SCORE) ln_w = w;
  else ln_w = log(w);  // w == 0 -> -inf (R13)
  const double gumbel = -log(-log(u));
  float f = (float)(ln_w + gumbel);  // one rounding fp64 -> fp32 (R15)
  f += 0.0f;                         // -0 -> +0 so that equal floats have equal bit patterns
  return ordermap(__float_as_uint(f));
}

__global__ void __launch_bounds__(256) nacl_keys_kernel(const float* __restrict__ imp, uint32_t* __restrict__ key,
                                                    int Hkv, int L, uint32_t k0, uint32_t k1, uint32_t layer, uint32_t flags) {
  const int p = blockIdx.y;  // b * Hkv + hk
  const int b = p / Hkv, hk = p - b * Hkv;
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= L) return;
  const size_t o = (size_t)p * L + j;
  key[o] = gumbel_key(imp[o], (uint32_t)j, (uint32_t)hk, (uint32_t)b, layer, k0, k1, flags);
}

// ------------------------------------------------------------------ block primitives
constexpr int ST = 1024;  // threads of the select CTA
constexpr int HB = 4096;  // histogram bins (12-bit first digit)

struct SelShared {
  uint32_t hist[HB];
  int warp_tot[32];
  int total;
  int bin, krem, cut;
};

// exclusive prefix sum of v over the block in thread order; total in `tot` (uniform)
__device__ __forceinline__ int block_excl_scan(int v, SelShared& sh, int& tot) {
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
template <class F>
__device__ void block_radix_select(F getval, int lo, int hi, int K, SelShared& sh, uint32_t& thr, int& cut) {
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
          if (above < krem && krem <= above + cnt[q]) { sh.bin = top - q; sh.krem = krem - above; sh.cut = cnt[q]; }
          above += cnt[q];
        }
      }
    }
    __syncthreads();
    prefix |= (uint32_t)sh.bin << shift;
    mask |= (uint32_t)(nb - 1) << shift;
    krem = sh.krem;
    n_eq = sh.cut;
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
      if (flag && running + excl + 1 == krem) sh.cut = j;
      __syncthreads();
      result = sh.cut;
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

// ------------------------------------------------------------------ cluster version
// Shared state of one CTA.  Every CTA counts its own slice into a histogram in its own shared memory (warp-
// aggregated), adds the non-empty bins to the head's histogram in global memory (L2 reductions; measured ~10x
// cheaper than exchanging whole histograms through distributed shared memory), and after ONE cluster barrier per
// radix pass every CTA reads the merged histogram back and finds the threshold bin itself.  Integer sums: exact
// and order-independent.  Each pass of each select has its own global histogram, cleared at kernel start.
struct ClShared {
  uint32_t hist[HB];
  int warp_tot[32];
  int total;
  int bin, krem, neq;   // result of a radix pass
  int cnt[3][8];        // per-rank counts: ties of select 0 / select 1, kept positions
  int cut[2];           // index of the last tie taken, select 0 / select 1
  int pad[2];           // sizeof % 16 == 0
};
static_assert(sizeof(ClShared) % 16 == 0, "the slices behind ClShared stay 16-byte aligned");
constexpr int kGhWordsPerSelect = 4096 + 1024 + 1024;  // global histogram words per select
constexpr int kGhWords = 2 * kGhWordsPerSelect;        // ... per head

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
// gh = this select's global histograms of the head (zero on entry); which = 0 / 1 (first / second select).
template <class F>
__device__ void cluster_radix_select(F getval, int nloc, int j0, int K, ClShared& sh, cg::cluster_group& cluster, uint32_t* gh,
                                     int which, uint32_t& thr, int& cut) {
  if (K <= 0) { thr = 0xFFFFFFFFu; cut = -1; return; }
  const unsigned rank = cluster.block_rank(), nrank = cluster.num_blocks();
  uint32_t prefix = 0, mask = 0;
  int krem = K, n_eq = 0;
#pragma unroll 1
  for (int pass = 0; pass < 3; ++pass) {
    const int shift = pass == 0 ? 20 : (pass == 1 ? 10 : 0);
    const int nb = pass == 0 ? 4096 : 1024;
    uint32_t* ghp = gh + (pass == 0 ? 0 : (pass == 1 ? 4096 : 5120));
    for (int i = threadIdx.x; i < nb; i += ST) sh.hist[i] = 0;
    __syncthreads();
    for (int base = 0; base < nloc; base += ST) {  // warp-uniform trip count
      const int i = base + (int)threadIdx.x;
      uint32_t v = 0;
      const bool take = i < nloc && getval(i, v) && (v & mask) == prefix;
      hist_add_aggregated(sh.hist, take, (v >> shift) & (uint32_t)(nb - 1));
    }
    __syncthreads();
    // thread t owns w consecutive bins, taken from the top: bins nb-1-t*w-(w-1) .. nb-1-t*w
    const int w = nb / ST;  // 4 or 1
    int cnt[4] = {0, 0, 0, 0}, sum = 0;
    const int top = nb - 1 - (int)threadIdx.x * w;
    if (nrank > 1) {
#pragma unroll
      for (int q = 0; q < 4; ++q)
        if (q < w) { const uint32_t h = sh.hist[top - q]; if (h) atomicAdd(&ghp[top - q], h); }
      __threadfence();
      cluster.sync();
#pragma unroll
      for (int q = 0; q < 4; ++q)
        if (q < w) cnt[q] = (int)__ldcg(&ghp[top - q]);
    } else {
#pragma unroll
      for (int q = 0; q < 4; ++q)
        if (q < w) cnt[q] = (int)sh.hist[top - q];
    }
#pragma unroll
    for (int q = 0; q < 4; ++q) sum += cnt[q];
    int tot;
    const int excl = cl_block_excl_scan(sum, sh, tot);
    if (excl < krem && krem <= excl + sum) {
      int above = excl;
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        if (q < w) {
          if (above < krem && krem <= above + cnt[q]) { sh.bin = top - q; sh.krem = krem - above; sh.neq = cnt[q]; }
          above += cnt[q];
        }
      }
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

#ifdef NACL_SEL_TRACE
__device__ long long g_sel_trace[16];
#define STAMP(k) if (blockIdx.x == 0 && threadIdx.x == 0) g_sel_trace[k] = clock64();
#else
#define STAMP(k)
#endif

// One cluster per (batch, kv head); CTA `rank` owns positions [rank*Lc, min(L, (rank+1)*Lc)).
// Dynamic shared memory: ClShared, uint32 ib[Lc] (order-mapped importance), uint32 kb[Lc] (order-mapped keys, later keep flags).
__global__ void __launch_bounds__(ST) nacl_select_cluster_kernel(const float* __restrict__ imp, int Hkv, int L, int Lc, int k1, int Br,
                                                                 int n_sink, int n_recent, int C, uint32_t sk0, uint32_t sk1,
                                                                 uint32_t layer, uint32_t flags, uint32_t* __restrict__ ghist,
                                                                 int32_t* __restrict__ out_idx) {
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

  STAMP(0)
  for (int i = threadIdx.x; i < nloc; i += ST) ib[i] = ordermap(__float_as_uint(row[i]));
  // this call's global histograms of the head: every CTA clears its share
  uint32_t* gh = ghist + (size_t)p * kGhWords;
  if (nrank > 1) {
    for (int i = (int)rank * ST + (int)threadIdx.x; i < kGhWords; i += (int)nrank * ST) gh[i] = 0;
    __threadfence();
  }
  cluster.sync();  // every CTA of the cluster is running and the global histograms are clear
  STAMP(1)
  auto free_pos = [&](int i) { const int j = j0 + i; return j >= lo && j < hi; };

  // a4: Proxy-Tokens Eviction, top-k1 of the importance outside the protected set
  uint32_t thr_p;
  int cut_p;
  cluster_radix_select([&](int i, uint32_t& v) { v = ib[i]; return free_pos(i); }, nloc, j0, k1, sh, cluster, gh, 0, thr_p, cut_p);
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
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int i = base + u * ST + (int)threadIdx.x;
        kk[u] = gumbel_key(i < nloc ? row[i] : 1.f, (uint32_t)(j0 + i), (uint32_t)hk, (uint32_t)b, layer, sk0, sk1, flags);
      }
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int i = base + u * ST + (int)threadIdx.x;
        if (i < nloc && free_pos(i) && !in_topk(i)) kb[i] = kk[u];
      }
    }
    __syncthreads();
  }
  STAMP(3)
  uint32_t thr_r;
  int cut_r;
  cluster_radix_select([&](int i, uint32_t& v) { if (!free_pos(i) || in_topk(i)) return false; v = kb[i]; return true; },
                       nloc, j0, Br, sh, cluster, gh + kGhWordsPerSelect, 1, thr_r, cut_r);

  STAMP(4)
  // a6: ascending kept-position list: keep flags, per-CTA counts, exclusive offsets over the cluster ranks, compaction
  int mine = 0;
  for (int i = threadIdx.x; i < nloc; i += ST) {
    int keep;
    if (!free_pos(i) || in_topk(i)) keep = 1;
    else { const uint32_t v = kb[i]; keep = (v > thr_r || (v == thr_r && j0 + i <= cut_r)) ? 1 : 0; }
    kb[i] = (uint32_t)keep;
    mine += keep;
  }
  int tot;
  cl_block_excl_scan(mine, sh, tot);
  if (threadIdx.x < nrank) cluster.map_shared_rank(&sh, threadIdx.x)->cnt[2][rank] = tot;
  cluster.sync();  // the last access to another CTA's shared memory lies before this barrier
  int running = 0;
  for (unsigned r = 0; r < rank; ++r) running += sh.cnt[2][r];
  int32_t* out = out_idx + (size_t)p * C;
#pragma unroll 1
  for (int base = 0; base < nloc; base += ST) {
    const int i = base + (int)threadIdx.x;
    const int keep = i < nloc ? (int)kb[i] : 0;
    int t2;
    const int excl = cl_block_excl_scan(keep, sh, t2);
    if (keep) {
      const int pos = running + excl;
      if (pos < C) out[pos] = j0 + i;
    }
    running += t2;
  }
  STAMP(5)
}

}  // namespace

cudaError_t launch_keys(const float* imp, uint32_t* key, int batch, int Hkv, int L, uint64_t seed, int layer,
                        uint32_t flags, cudaStream_t st) {
  dim3 grid((L + 255) / 256, batch * Hkv);
  nacl_keys_kernel<<<grid, 256, 0, st>>>(imp, key, Hkv, L, (uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32),
                                    (uint32_t)layer, flags);
  return cudaGetLastError();
}

// slices of at most this many positions per CTA stay in shared memory (2 x 4 bytes each)
constexpr int kMaxSlice = 20480;

bool select_uses_cluster(int L) { return (L + 7) / 8 <= kMaxSlice; }

cudaError_t launch_select(const float* imp, uint32_t* key, int batch, int Hkv, int L, int budget_proxy, int budget_random,
                          int n_sink, int n_recent, uint64_t seed, int layer, uint32_t flags, int32_t* out_idx,
                          cudaStream_t st) {
  const int C = budget_proxy + budget_random;
  if (C == 0) return cudaSuccess;
  const int k1 = budget_proxy - n_sink - n_recent;
  const uint32_t sk0 = (uint32_t)(seed & 0xFFFFFFFFu), sk1 = (uint32_t)(seed >> 32);
  if (!select_uses_cluster(L)) {
    // very long rows: sampling keys in a kernel of their own, one CTA per head working out of global memory
    if (budget_random > 0) {
      StageScope sc(ST_KEYS, st);
      cudaError_t e = launch_keys(imp, key, batch, Hkv, L, seed, layer, flags, st);
      if (e != cudaSuccess) return e;
    }
    StageScope sc(ST_SELECT, st);
    nacl_select_kernel<<<batch * Hkv, ST, 0, st>>>(imp, key, L, k1, budget_random, n_sink, n_recent, C, out_idx);
    return cudaGetLastError();
  }
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
  int n = 0, Lc = 0;
  size_t dyn = 0;
  double best = 0.0;
  cudaError_t e = cudaFuncSetAttribute(nacl_select_cluster_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       (int)(sizeof(ClShared) + (size_t)kMaxSlice * 2 * sizeof(uint32_t)));
  if (e != cudaSuccess) return e;
  for (int c = 1; c <= 8; c *= 2) {
    const int lc = ((L + c - 1) / c + 3) / 4 * 4;
    if (lc > kMaxSlice) continue;
    if (c > 1 && L / c < ST / 2) break;  // slices below half a block of positions are not worth a barrier per pass
    const size_t d = sizeof(ClShared) + (size_t)lc * 2 * sizeof(uint32_t);
    static int active_cache[4][2] = {{0, 0}, {0, 0}, {0, 0}, {0, 0}};  // [log2 c][smem class]: co-resident clusters
    const int ci = c == 1 ? 0 : (c == 2 ? 1 : (c == 4 ? 2 : 3)), si = d > 100 * 1024 ? 1 : 0;
    int active = active_cache[ci][si];
    if (active == 0) {
      cfg.gridDim = dim3((unsigned)(c * 64));
      cfg.dynamicSmemBytes = si ? sizeof(ClShared) + (size_t)kMaxSlice * 2 * sizeof(uint32_t) : 100 * 1024;
      attr[0].val.clusterDim.x = (unsigned)c;
      if (cudaOccupancyMaxActiveClusters(&active, nacl_select_cluster_kernel, &cfg) != cudaSuccess || active < 1) {
        cudaGetLastError();
        active = kNumSMs / c / 2;  // conservative guess
      }
      active_cache[ci][si] = active;
    }
    const double waves = (double)((heads + active - 1) / active);
    const double cost = waves * (37000.0 + 6.0 * lc);
    if (n == 0 || cost < best) { n = c; Lc = lc; dyn = d; best = cost; }
  }
  if (n == 0) return cudaErrorInvalidConfiguration;
  cfg.gridDim = dim3((unsigned)(heads * n));
  cfg.dynamicSmemBytes = dyn;
  attr[0].val.clusterDim.x = (unsigned)n;
  StageScope sc(ST_SELECT, st);
  return cudaLaunchKernelEx(&cfg, nacl_select_cluster_kernel, imp, Hkv, L, Lc, k1, budget_random, n_sink, n_recent, C, sk0, sk1,
                            (uint32_t)layer, flags, key /* scratch: global histograms */, out_idx);
}

// 4-byte words of the `key` scratch the select needs (cluster path: global histograms; long-row path: the keys)
size_t select_scratch_words(int batch, int Hkv, int L) {
  if (!select_uses_cluster(L)) return (size_t)batch * Hkv * L;
  return (size_t)batch * Hkv * kGhWords;
}

}  // namespace nacl

#ifdef NACL_SEL_TRACE
extern "C" __attribute__((visibility("default"))) int nacl_debug_sel_trace_read(long long* host) {
  return (int)cudaMemcpyFromSymbol(host, nacl::g_sel_trace, sizeof(nacl::g_sel_trace));
}
#endif
