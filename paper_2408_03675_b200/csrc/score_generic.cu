// score_generic.cu -- CUDA-core scoring kernels (steps a1-a3 of SURVEY.md section 8) for every
// shape the tensor-core path does not take: fp32 inputs (config 1), d != 128, odd G*P.
//
//   stats   : per proxy row and L-chunk, (m, Z) = (max_j s, sum_j exp(s - m))
//   combine : lse_i = m_i + ln Z_i, merged over the chunks in ascending order
//   colsum  : imp[j] = sum_{g,i} exp(s[i,j] - lse_i)
// with s[i,j] = Q[i,:].K[j,:] / sqrt(d) in fp32 FMAs, ascending t, so both
// sweeps see bit-identical logits.  No floating-point atomics: every sum has a fixed order.
#include "nacl_internal.cuh"

namespace nacl {
namespace {

constexpr int TK = 64;        // keys per tile
constexpr int RB = 64;        // proxy rows per batch
constexpr int NT = 256;       // threads per block
constexpr int SUB = NT / 64;  // 4 interleaved subsets of the "other" dimension
constexpr int U = 16;         // (64 / SUB) items of the other dimension per thread

__device__ __forceinline__ float to_float(float v) { return v; }
__device__ __forceinline__ float to_float(__nv_bfloat16 v) { return __bfloat162float(v); }

// rows [row0, row0+n_valid) of a [*, d] matrix -> smem [64][d+1] as fp32, zero rows beyond n_valid
// (rs = elements between consecutive rows of src)
template <typename T>
__device__ __forceinline__ void stage_rows(const T* __restrict__ src, int n_valid, int d, float* dst, long long rs) {
  const int ld = d + 1;
  for (int e = threadIdx.x; e < 64 * d; e += NT) {
    int r = e / d, t = e - r * d;
    dst[r * ld + t] = r < n_valid ? to_float(src[(size_t)r * rs + t]) : 0.f;
  }
}

// a[u] = own[own_idx,:] . other[sub + SUB*u,:]   (ascending t, fp32 FMA)
__device__ __forceinline__ void dots(const float* own, int own_idx, const float* other, int sub, int d, float (&a)[U]) {
  const int ld = d + 1;
  const float* o = own + own_idx * ld;
  const float* x = other + sub * ld;
#pragma unroll
  for (int u = 0; u < U; ++u) a[u] = 0.f;
  for (int t = 0; t < d; ++t) {
    float ov = o[t];
#pragma unroll
    for (int u = 0; u < U; ++u) a[u] = fmaf(ov, x[u * SUB * ld + t], a[u]);
  }
}

// global row index of proxy row gr (0..rows) of kv head hk:  [batch, Hq, P] flattened
__device__ __forceinline__ size_t row_id(int b, int hk, int gr, int G, int P, int Hq) {
  int g = gr / P, i = gr - g * P;
  return ((size_t)b * Hq + (size_t)hk * G + g) * P + i;
}

template <typename T>
__global__ void __launch_bounds__(NT) nacl_stats_kernel(const T* __restrict__ K, const T* __restrict__ Q, float2* __restrict__ part,
                                                    int L, int Hq, int Hkv, int d, int P, int G, int chunk, int n_chunks,
                                                    float inv_sqrt_d, int causal, long long sb, long long sh, long long sr) {
  extern __shared__ float smem[];
  const int ld = d + 1;
  float* Qs = smem;            // [64][d+1]
  float* Ks = smem + 64 * ld;  // [64][d+1]
  __shared__ float2 red[SUB][RB];
  const int c = blockIdx.x, hk = blockIdx.y, b = blockIdx.z;
  const int rows = G * P;
  const int j_begin = c * chunk, j_end = min(L, j_begin + chunk);
  const T* Kh = K + (size_t)b * sb + (size_t)hk * sh;
  const T* Qh = Q + ((size_t)b * Hq + (size_t)hk * G) * (size_t)P * d;  // the group's G*P rows are contiguous
  const int r = threadIdx.x & 63, sub = threadIdx.x >> 6;

  for (int rb = 0; rb < rows; rb += RB) {
    const int nr = min(RB, rows - rb);
    __syncthreads();
    stage_rows(Qh + (size_t)rb * d, nr, d, Qs, d);
    float m = -INFINITY, z = 0.f;
    for (int j0 = j_begin; j0 < j_end; j0 += TK) {
      const int nk = min(TK, j_end - j0);
      __syncthreads();
      stage_rows(Kh + (size_t)j0 * sr, nk, d, Ks, sr);
      __syncthreads();
      float a[U];
      dots(Qs, r, Ks, sub, d, a);
#pragma unroll
      for (int u = 0; u < U; ++u) {
        // NACL_FLAG_CAUSAL (R1): proxy row i is prompt position L-P+i and sees keys j <= L-P+i
        const int jj = j0 + sub + SUB * u;
        if (sub + SUB * u < nk && !(causal && jj > L - P + (rb + r) % P)) {
          float x = a[u] * inv_sqrt_d;
          if (x > m) { z = z * expf(m - x) + 1.f; m = x; }
          else z += expf(x - m);
        }
      }
    }
    red[sub][r] = make_float2(m, z);
    __syncthreads();
    if (sub == 0 && r < nr) {
      float mm = red[0][r].x, zz = red[0][r].y;
#pragma unroll
      for (int s2 = 1; s2 < SUB; ++s2) merge_mz(mm, zz, red[s2][r].x, red[s2][r].y);
      part[row_id(b, hk, rb + r, G, P, Hq) * n_chunks + c] = make_float2(mm, zz);
    }
  }
}

__global__ void nacl_combine_kernel(const float2* __restrict__ part, float* __restrict__ lse, float* __restrict__ lse_out,
                               int n_rows, int n_chunks) {
  int row = blockIdx.x * blockDim.x + threadIdx.x;
  if (row >= n_rows) return;
  float m = -INFINITY, z = 0.f;
  for (int c = 0; c < n_chunks; ++c) {
    float2 p = part[(size_t)row * n_chunks + c];
    merge_mz(m, z, p.x, p.y);
  }
  float v = m + logf(z);
  lse[row] = v;
  if (lse_out) lse_out[row] = v;
}

template <typename T>
__global__ void __launch_bounds__(NT) nacl_colsum_kernel(const T* __restrict__ K, const T* __restrict__ Q, const float* __restrict__ lse,
                                                     float* __restrict__ imp, float* __restrict__ imp_out,
                                                     int L, int Hq, int Hkv, int d, int P, int G, float inv_sqrt_d, int causal,
                                                     long long sb, long long sh, long long sr) {
  extern __shared__ float smem[];
  const int ld = d + 1;
  float* Qs = smem;
  float* Ks = smem + 64 * ld;
  __shared__ float lse_s[RB];
  __shared__ float red[SUB][TK];
  const int hk = blockIdx.y, b = blockIdx.z;
  const int rows = G * P;
  const int j0 = blockIdx.x * TK;
  const int nk = min(TK, L - j0);
  const T* Kh = K + (size_t)b * sb + (size_t)hk * sh;
  const T* Qh = Q + ((size_t)b * Hq + (size_t)hk * G) * (size_t)P * d;
  const int j = threadIdx.x & 63, sub = threadIdx.x >> 6;

  stage_rows(Kh + (size_t)j0 * sr, nk, d, Ks, sr);
  float acc = 0.f;
  for (int rb = 0; rb < rows; rb += RB) {
    const int nr = min(RB, rows - rb);
    __syncthreads();
    stage_rows(Qh + (size_t)rb * d, nr, d, Qs, d);
    if (threadIdx.x < RB) lse_s[threadIdx.x] = threadIdx.x < nr ? lse[row_id(b, hk, rb + threadIdx.x, G, P, Hq)] : 0.f;
    __syncthreads();
    float a[U];
    dots(Ks, j, Qs, sub, d, a);
#pragma unroll
    for (int u = 0; u < U; ++u) {
      int rr = sub + SUB * u;
      if (rr < nr && !(causal && j0 + j > L - P + (rb + rr) % P)) acc += expf(a[u] * inv_sqrt_d - lse_s[rr]);
    }
  }
  red[sub][j] = acc;
  __syncthreads();
  if (sub == 0 && j < nk) {
    float v = red[0][j];
#pragma unroll
    for (int s2 = 1; s2 < SUB; ++s2) v += red[s2][j];
    size_t o = ((size_t)b * Hkv + hk) * (size_t)L + j0 + j;
    imp[o] = v;
    if (imp_out) imp_out[o] = v;
  }
}

template <typename T>
cudaError_t launch_typed(const Shape& s, const void* K, const void* Q, const SplitPlan& sp, const Workspace& ws,
                         const float* lse_in, bool causal, float* imp_out, float* lse_out, cudaStream_t st, bool stats_only) {
  if (stats_only && (!lse_out || lse_in)) return cudaErrorInvalidValue;
  const size_t smem = (size_t)2 * 64 * (s.d + 1) * sizeof(float);
  cudaError_t e;
  if ((e = cudaFuncSetAttribute(nacl_stats_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)) != cudaSuccess) return e;
  if ((e = cudaFuncSetAttribute(nacl_colsum_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)) != cudaSuccess) return e;
  const float inv_sqrt_d = 1.0f / sqrtf((float)s.d);
  dim3 g1(sp.n_chunks, s.Hkv, s.batch);
  const int n_rows = s.batch * s.Hq * s.P;
  const float* lse = ws.lse;
  if (lse_in) {  // the caller has the row statistics: no sweep S
    lse = lse_in;
    if (lse_out && (e = cudaMemcpyAsync(lse_out, lse_in, (size_t)n_rows * sizeof(float), cudaMemcpyDeviceToDevice, st)) != cudaSuccess)
      return e;
  } else {
  {
    StageScope sc(ST_STATS, st);
    nacl_stats_kernel<T><<<g1, NT, smem, st>>>((const T*)K, (const T*)Q, ws.part, s.L, s.Hq, s.Hkv, s.d, s.P, s.G, sp.chunk,
                                          sp.n_chunks, inv_sqrt_d, causal ? 1 : 0, s.kv_sb, s.kv_sh, s.kv_sr);
  }
  if ((e = cudaGetLastError()) != cudaSuccess) return e;
  {
    StageScope sc(ST_COMBINE, st);
    nacl_combine_kernel<<<(n_rows + 127) / 128, 128, 0, st>>>(ws.part, ws.lse, lse_out, n_rows, sp.n_chunks);
  }
  if ((e = cudaGetLastError()) != cudaSuccess) return e;
  }
  if (stats_only) return cudaSuccess;
  dim3 g2((s.L + TK - 1) / TK, s.Hkv, s.batch);
  {
    StageScope sc(ST_COLSUM, st);
    nacl_colsum_kernel<T><<<g2, NT, smem, st>>>((const T*)K, (const T*)Q, lse, ws.imp, imp_out, s.L, s.Hq, s.Hkv, s.d, s.P,
                                           s.G, inv_sqrt_d, causal ? 1 : 0, s.kv_sb, s.kv_sh, s.kv_sr);
  }
  return cudaGetLastError();
}

}  // namespace

cudaError_t launch_score_generic(const Shape& s, const void* K, const void* Q, const SplitPlan& sp, const Workspace& ws,
                                 const float* lse_in, bool causal, float* imp_out, float* lse_out, cudaStream_t st, bool stats_only) {
  if (s.dtype == NACL_DTYPE_F32) return launch_typed<float>(s, K, Q, sp, ws, lse_in, causal, imp_out, lse_out, st, stats_only);
  return launch_typed<__nv_bfloat16>(s, K, Q, sp, ws, lse_in, causal, imp_out, lse_out, st, stats_only);
}

}  // namespace nacl
