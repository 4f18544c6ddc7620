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
// Integer work only after the keys: results are bit-exact functions of (imp, key).
#include "nacl_internal.cuh"

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

__global__ void __launch_bounds__(256) nacl_keys_kernel(const float* __restrict__ imp, uint32_t* __restrict__ key,
                                                    int Hkv, int L, uint32_t k0, uint32_t k1, uint32_t layer, uint32_t flags) {
  const int p = blockIdx.y;  // b * Hkv + hk
  const int b = p / Hkv, hk = p - b * Hkv;
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= L) return;
  const size_t o = (size_t)p * L + j;
  const uint32_t x = philox4x32_10_word0((uint32_t)j, (uint32_t)hk, (uint32_t)b, layer, k0, k1);
  const double u = ((double)(x >> 9) + 0.5) * 0x1p-23;  // exact; u in [2^-24, 1-2^-24]
  const double w = (double)imp[o];
  double ln_w;
  if (flags & NACL_FLAG_SAMPLE_UNIFORM) ln_w = 0.0;
  else if (flags & NACL_FLAG_SAMPLE_SOFTMAX_OF_SCORE) ln_w = w;
  else ln_w = log(w);  // w == 0 -> -inf (R13)
  const double gumbel = -log(-log(u));
  float f = (float)(ln_w + gumbel);  // one rounding fp64 -> fp32 (R15)
  f += 0.0f;                         // -0 -> +0 so that equal floats have equal bit patterns
  key[o] = ordermap(__float_as_uint(f));
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
    for (int j = lo + (int)threadIdx.x; j < hi; j += ST) {
      uint32_t v;
      if (getval(j, v) && (v & mask) == prefix) atomicAdd(&sh.hist[(v >> shift) & (uint32_t)(nb - 1)], 1u);
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

}  // namespace

cudaError_t launch_keys(const float* imp, uint32_t* key, int batch, int Hkv, int L, uint64_t seed, int layer,
                        uint32_t flags, cudaStream_t st) {
  dim3 grid((L + 255) / 256, batch * Hkv);
  nacl_keys_kernel<<<grid, 256, 0, st>>>(imp, key, Hkv, L, (uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32),
                                    (uint32_t)layer, flags);
  return cudaGetLastError();
}

cudaError_t launch_select(const float* imp, const uint32_t* key, int batch, int Hkv, int L, int budget_proxy,
                          int budget_random, int n_sink, int n_recent, int32_t* out_idx, cudaStream_t st) {
  const int C = budget_proxy + budget_random;
  if (C == 0) return cudaSuccess;
  const int k1 = budget_proxy - n_sink - n_recent;
  nacl_select_kernel<<<batch * Hkv, ST, 0, st>>>(imp, key, L, k1, budget_random, n_sink, n_recent, C, out_idx);
  return cudaGetLastError();
}

}  // namespace nacl
