// gather.cu -- step a7 of SURVEY.md section 8: cache compaction K,V <- K_S,V_S.
// Pure data movement, bit-exact rows.  Every thread moves 16-byte vectors (LDG.128 / STG.128):
// consecutive threads take consecutive vectors of the OUTPUT, so writes are fully coalesced and
// reads are whole contiguous rows (row_bytes >= 128 B in every supported shape) at ascending
// addresses.  Inputs are streamed past L1 (read once); outputs are streaming stores.
#include "nacl_internal.cuh"

namespace nacl {
namespace {

__device__ __forceinline__ int4 ld_stream(const int4* p) {
  int4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.s32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
  return r;
}
__device__ __forceinline__ void st_stream(int4* p, const int4& v) {
  asm volatile("st.global.L1::no_allocate.v4.s32 [%0], {%1,%2,%3,%4};" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}

constexpr int GT = 256;  // threads per block
constexpr int GU = 4;    // vectors of K and of V in flight per thread

// vpr = 16-byte vectors per row; n_vec = n_prob * C * vpr output vectors per tensor.  Strides in 16-byte vectors:
// (sb, sh, sr) of K/V per batch element / kv head / row, (ob, oh, orow) of the outputs.
// Paged source (table != nullptr): row j of batch element b = row j % ps of page table[b * tstride + j / ps], page stride sp.
struct GatherLayout { long long sb, sh, sr, ob, oh, orow; int Hkv; const int32_t* table; int ps, tstride; long long sp; };
__global__ void __launch_bounds__(GT) nacl_gather_kernel(const int4* __restrict__ K, const int4* __restrict__ V,
                                                     const int32_t* __restrict__ idx, int C, int vpr, GatherLayout ly,
                                                     size_t n_vec, int4* __restrict__ oK, int4* __restrict__ oV) {
  const size_t stride = (size_t)gridDim.x * GT;
  for (size_t v0 = (size_t)blockIdx.x * GT + threadIdx.x; v0 < n_vec; v0 += stride * GU) {
    size_t src[GU], dst[GU];
    bool ok[GU];
#pragma unroll
    for (int u = 0; u < GU; ++u) {
      const size_t v = v0 + (size_t)u * stride;
      ok[u] = v < n_vec;
      if (ok[u]) {
        const size_t row = v / (size_t)vpr;          // p * C + c
        const int off = (int)(v - row * (size_t)vpr);
        const size_t p = row / (size_t)C;
        const int c = (int)(row - p * (size_t)C);
        const int b = (int)(p / (size_t)ly.Hkv), hk = (int)(p - (size_t)b * ly.Hkv);
        const int j = idx[row];
        if (ly.table) {
          const long long pg = __ldg(&ly.table[(size_t)b * ly.tstride + j / ly.ps]);
          src[u] = (size_t)(pg * ly.sp + hk * ly.sh + (long long)(j % ly.ps) * ly.sr) + off;
        } else {
          src[u] = (size_t)(b * ly.sb + hk * ly.sh + (long long)j * ly.sr) + off;
        }
        dst[u] = (size_t)(b * ly.ob + hk * ly.oh + (long long)c * ly.orow) + off;
      }
    }
    int4 a[GU], b4[GU];
#pragma unroll
    for (int u = 0; u < GU; ++u)
      if (ok[u]) { a[u] = ld_stream(K + src[u]); b4[u] = ld_stream(V + src[u]); }
#pragma unroll
    for (int u = 0; u < GU; ++u)
      if (ok[u]) {
        st_stream(oK + dst[u], a[u]);
        st_stream(oV + dst[u], b4[u]);
      }
  }
}

__global__ void __launch_bounds__(256) nacl_compose_positions_kernel(const int32_t* __restrict__ pos_in, long long in_stride,
                                                                     const int32_t* __restrict__ idx, int C,
                                                                     int32_t* __restrict__ pos_out, long long out_stride) {
  const int p = blockIdx.y;
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= C) return;
  pos_out[(size_t)p * out_stride + c] = pos_in[(size_t)p * in_stride + idx[(size_t)p * C + c]];
}

// ---- small helpers of the selection variants
__global__ void __launch_bounds__(256) nacl_head_sum_kernel(const float* __restrict__ imp, float* __restrict__ out, int Hkv, int L) {
  const int b = blockIdx.y;
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= L) return;
  float a = 0.f;
  for (int hk = 0; hk < Hkv; ++hk) a = __fadd_rn(a, imp[((size_t)b * Hkv + hk) * L + j]);  // head order, no contraction
  out[(size_t)b * L + j] = a;
}
__global__ void __launch_bounds__(256) nacl_replicate_idx_kernel(const int32_t* __restrict__ shared, int32_t* __restrict__ idx,
                                                                 int Hkv, int C) {
  const int b = blockIdx.y;
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= C) return;
  const int32_t v = shared[(size_t)b * C + c];
  for (int hk = 0; hk < Hkv; ++hk) idx[((size_t)b * Hkv + hk) * C + c] = v;
}
__global__ void __launch_bounds__(256) nacl_protect_kernel(float* __restrict__ imp, int L, const int32_t* __restrict__ protect_idx,
                                                           int n_protect) {
  const int e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= n_protect) return;
  const int j = protect_idx[e];
  if (j >= 0 && j < L) imp[(size_t)blockIdx.y * L + j] = __int_as_float(0x7F800000);
}

}  // namespace

cudaError_t launch_head_sum(const float* imp, float* out, int batch, int Hkv, int L, cudaStream_t st) {
  nacl_head_sum_kernel<<<dim3((L + 255) / 256, batch), 256, 0, st>>>(imp, out, Hkv, L);
  return cudaGetLastError();
}
cudaError_t launch_replicate_idx(const int32_t* shared, int32_t* idx, int batch, int Hkv, int C, cudaStream_t st) {
  if (C == 0) return cudaSuccess;
  nacl_replicate_idx_kernel<<<dim3((C + 255) / 256, batch), 256, 0, st>>>(shared, idx, Hkv, C);
  return cudaGetLastError();
}
cudaError_t launch_protect(float* imp, int n_prob, int L, const int32_t* protect_idx, int n_protect, cudaStream_t st) {
  if (n_protect == 0) return cudaSuccess;
  nacl_protect_kernel<<<dim3((n_protect + 255) / 256, n_prob), 256, 0, st>>>(imp, L, protect_idx, n_protect);
  return cudaGetLastError();
}

cudaError_t launch_gather(const void* K, const void* V, const int32_t* idx, const Shape& s, int C, int row_bytes,
                          void* out_K, void* out_V, cudaStream_t st) {
  const int vpr = row_bytes / 16;
  const size_t n_vec = (size_t)s.batch * s.Hkv * C * vpr;
  if (n_vec == 0) return cudaSuccess;
  const long long epv = 16 / s.esize;  // elements per 16-byte vector (strides are multiples of it)
  const GatherLayout ly{s.kv_sb / epv, s.kv_sh / epv, s.kv_sr / epv, s.o_sb / epv, s.o_sh / epv, s.o_sr / epv, s.Hkv,
                        s.table, s.ps, s.tstride, s.kv_sp / epv};
  size_t want = (n_vec + (size_t)GT * GU - 1) / ((size_t)GT * GU);
  const size_t cap = (size_t)kNumSMs * 8 * 4;  // a few waves of 8 resident CTAs per SM
  int blocks = (int)(want < cap ? want : cap);
  nacl_gather_kernel<<<blocks, GT, 0, st>>>((const int4*)K, (const int4*)V, idx, C, vpr, ly, n_vec, (int4*)out_K, (int4*)out_V);
  return cudaGetLastError();
}

cudaError_t launch_compose_positions(const int32_t* pos_in, long long in_stride, const int32_t* idx, int n_prob, int C,
                                     int32_t* pos_out, long long out_stride, cudaStream_t st) {
  if (C == 0 || n_prob == 0) return cudaSuccess;
  nacl_compose_positions_kernel<<<dim3((C + 255) / 256, n_prob), 256, 0, st>>>(pos_in, in_stride, idx, C, pos_out, out_stride);
  return cudaGetLastError();
}

}  // namespace nacl
