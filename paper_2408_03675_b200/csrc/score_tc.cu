// score_tc.cu -- tensor-core scoring path: steps a1-a3 of SURVEY.md section 8 in ONE persistent,
// warp-specialised sm_100a kernel (tcgen05.mma + TMEM accumulators + TMA-staged tiles).
//
//   a1  s[i,j] = Q[i,:].K[j,:] / sqrt(d)                      PAPER.md:59, Alg.1
//   a2  lse_i  = log sum_j exp(s[i,j])   (full-length softmax)
//   a3  imp[j] = sum_{g,i} exp(s[i,j] - lse_i)
//
// Serves bf16, d == 128, G*P a multiple of 16 and <= 256.  Everything else takes score_generic.cu.
//
// Work decomposition.  The logits are never written to memory, and the column sum needs the
// complete row normaliser first, so every key tile is scored twice: an S item (softmax
// statistics) and a C item (column sum).  An item is (phase, kv head, chunk of `chunk` keys).
// Items are handed out through one atomic ticket in the order
//     S(0) .. S(D-1), S(D), C(0), S(D+1), C(1), ...                       (D = lag in heads)
// so that the second read of a head's K tiles follows the first one by a few heads and is served
// by the 126 MB L2 instead of HBM.  C(h) needs lse of head h: the CTA that finishes the last S
// item of a head (a counter per head) merges the per-chunk partials in ascending chunk order and
// publishes lse with a release flag; C items acquire it.  A C item's ticket is larger than the
// tickets of all S items it waits for, and S items wait for nothing, so the wait cannot deadlock.
// No floating-point atomics anywhere: all sums have a fixed order (deterministic).
//
// Two MMA orientations share the same shared-memory operands (both K-major, 128B swizzle):
//   S items:  D[row, key] = Q_half (M=128 proxy rows) x K_tile^T (N=128 keys)   -> a thread owns a
//             proxy row, its running (max, sum-exp) live in two registers;
//   C items:  D[key, row] = K_tile (M=128 keys) x Q^T (N = G*P proxy rows)       -> a thread owns a
//             key, its column sum is a private register, no cross-thread reduction.
//
// Warp roles (320 threads, 1 CTA per SM): warps 0-7 = two epilogue warpgroups (warp%4 = TMEM lane
// quarter; warpgroup w drains TMEM buffer w, i.e. every other tile), warp 8 = ticket + TMA
// producer, warp 9 = TMEM allocator + tcgen05.mma issuer.
#include <cuda.h>

#include "nacl_internal.cuh"

namespace nacl {
namespace {

constexpr int TILE = 128;                      // keys per tile
constexpr int HD = 128;                        // head dim served by this path
constexpr int BOX_BYTES = 128 * 128;           // one TMA box: 128 rows x 64 bf16 (128 B, swizzled)
constexpr int KSTAGE_BYTES = 2 * BOX_BYTES;    // a K tile = two boxes (d 0..63, d 64..127)
constexpr int N_EPI_WARPS = 8;
constexpr int EPI_THREADS = N_EPI_WARPS * 32;
constexpr int W_TMA = 8, W_MMA = 9, W_AUX = 11;  // warp roles after the 8 epilogue warps: TMA, MMA issuers 9 and 10 (one per warpgroup), helper
constexpr int NTHREADS = EPI_THREADS + 4 * 32;
constexpr int RING = 4;                        // ticket ring slots
constexpr int TMEM_COLS = 512;
constexpr int N_BUFS = 4;                      // TMEM accumulator buffers, two per epilogue warpgroup
constexpr int BUF_COLS = 128;                  // TMEM columns per accumulator buffer
constexpr uint32_t SPIN_LIMIT = 1u << 24;      // watchdog: a wait that long is a bug -> trap (loud failure)

// Optional wait/compute cycle accounting per warp role (diagnostics build only: -DNACL_TC_TRACE).
#ifdef NACL_TC_TRACE
#define TR_N 16
__device__ long long g_trace[160][12][TR_N];
#define TR_DECL long long tr_[TR_N]; for (int i_ = 0; i_ < TR_N; ++i_) tr_[i_] = 0; const long long tr_start_ = clock64();
#define TRW(cat, ...) { const long long t_ = clock64(); __VA_ARGS__; tr_[cat] += clock64() - t_; }
#define TR_FLUSH() { tr_[15] = clock64() - tr_start_; if (lane == 0 && blockIdx.x < 160) for (int i_ = 0; i_ < TR_N; ++i_) g_trace[blockIdx.x][warp][i_] = tr_[i_]; }
#else
#define TR_DECL
#define TRW(cat, ...) { __VA_ARGS__; }
#define TR_FLUSH()
#endif

struct TcParams {
  int L, rows, n_halves, n_chunks, tiles_per_chunk, total_tiles;
  int heads, lag, n_items;
  int n_slots;        // partials per (row, chunk): 2 when both warpgroups see every proxy row (rows <= 128), else 1
  float scale_log2;   // log2(e) / sqrt(d)
  int* ticket;        // [1]
  int* cnt;           // [heads]  finished S items per head
  int* flag;          // [heads]  1 once lse of the head is published
  float2* part;       // [heads, n_chunks, 2, rows]  (m, z) per chunk and epilogue warpgroup, log2 domain
  float* lse2;        // [heads*rows]            log2-domain LSE
  float* lse_out;     // optional, natural log
  float* imp;         // [heads, L]
  float* imp_out;     // optional
};

// ------------------------------------------------------------------ PTX wrappers
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t a, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(a), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t a) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(a) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t a, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(a), "r"(bytes) : "memory");
}
__device__ __forceinline__ uint32_t mbar_try_wait(uint32_t a, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
      "selp.u32 %0, 1, 0, p;\n\t}"
      : "=r"(ok)
      : "r"(a), "r"(parity)
      : "memory");
  return ok;
}
__device__ __forceinline__ void mbar_wait(uint32_t a, uint32_t parity) {
  uint32_t spins = 0;
  while (!mbar_try_wait(a, parity))
    if (++spins > SPIN_LIMIT) __trap();
}

__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* tm, int c0, int c1, uint32_t bar) {
  asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
               ::"r"(dst), "l"(tm), "r"(c0), "r"(c1), "r"(bar)
               : "memory");
}
__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap* tm, int c0, int c1, int c2, uint32_t bar) {
  asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
               ::"r"(dst), "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(bar)
               : "memory");
}

__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
// D[tmem] (+)= A[smem] * B[smem]^T, bf16 inputs, fp32 accumulate; issued by ONE thread
__device__ __forceinline__ void tc_mma(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
      ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
      : "memory");
}
// waits for this thread's TMEM loads; the registers are in/out operands so that no use of them is scheduled above the wait
__device__ __forceinline__ void tc_wait_ld(uint32_t (&v)[32]) {
  asm volatile("tcgen05.wait::ld.sync.aligned;"
               : "+r"(v[0]), "+r"(v[1]), "+r"(v[2]), "+r"(v[3]), "+r"(v[4]), "+r"(v[5]), "+r"(v[6]), "+r"(v[7]), "+r"(v[8]),
                 "+r"(v[9]), "+r"(v[10]), "+r"(v[11]), "+r"(v[12]), "+r"(v[13]), "+r"(v[14]), "+r"(v[15]), "+r"(v[16]),
                 "+r"(v[17]), "+r"(v[18]), "+r"(v[19]), "+r"(v[20]), "+r"(v[21]), "+r"(v[22]), "+r"(v[23]), "+r"(v[24]),
                 "+r"(v[25]), "+r"(v[26]), "+r"(v[27]), "+r"(v[28]), "+r"(v[29]), "+r"(v[30]), "+r"(v[31])
               :
               : "memory");
}

// 32 lanes x 32 consecutive columns: thread t of the warp receives lane (quarter*32 + t), columns c..c+31
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&v)[32]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
      "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
      : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
        "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]),
        "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]),
        "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
      : "r"(taddr)
      : "memory");
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&v)[32]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
      : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
        "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
      : "r"(taddr)
      : "memory");
}

__device__ __forceinline__ float fast_exp2(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

__device__ __forceinline__ int ld_acquire(const int* p) {
  int v;
  asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_release(int* p, int v) {
  asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

__device__ __forceinline__ uint32_t lds_acquire(uint32_t a) {
  uint32_t v;
  asm volatile("ld.acquire.cta.shared::cta.u32 %0, [%1];" : "=r"(v) : "r"(a) : "memory");
  return v;
}
__device__ __forceinline__ void sts_release(uint32_t a, uint32_t v) {
  asm volatile("st.release.cta.shared::cta.u32 [%0], %1;" ::"r"(a), "r"(v) : "memory");
}

// lse of one proxy row from its per-(chunk, warpgroup) partials pp[c * stride], c < np, merged in ascending order with
// 16 loads in flight.  Consecutive lanes own consecutive rows, so every load of the warp is one contiguous 256 B.
__device__ __noinline__ float merge_row(const float2* __restrict__ pp, int np, size_t stride) {
  float m = -INFINITY, z = 0.f;
  for (int c0 = 0; c0 < np; c0 += 16) {
    float2 a[16];
#pragma unroll
    for (int e = 0; e < 16; ++e) {
      a[e] = __ldcg(&pp[(size_t)(c0 + e < np ? c0 + e : np - 1) * stride]);
      if (c0 + e >= np) a[e] = make_float2(-INFINITY, 0.f);
    }
    float mn = m;
#pragma unroll
    for (int e = 0; e < 16; ++e) mn = fmaxf(mn, a[e].x);
    if (mn != -INFINITY) {
      float acc = z * exp2f(m - mn);
#pragma unroll
      for (int e = 0; e < 16; ++e) acc += a[e].y * exp2f(a[e].x - mn);
      z = acc;
      m = mn;
    }
  }
  return m + log2f(z);
}

// K-major operand tile, 128-byte swizzle, rows of 128 B, 8-row groups 1024 B apart (sm_100 descriptor v1)
__device__ __forceinline__ uint64_t umma_desc(uint32_t smem_addr) {
  return (uint64_t)((smem_addr >> 4) & 0x3FFFu) | (1ull << 16) | (64ull << 32) | (1ull << 46) | (2ull << 61);
}
// kind::f16 instruction descriptor: D fp32, A/B bf16, both K-major
__device__ __forceinline__ uint32_t umma_idesc(int M, int N) {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}

struct Item { int phase, head, tile0, ntiles, chunk; };  // phase 0 = S (statistics), 1 = C (column sum)

__device__ __forceinline__ Item decode_item(int t, const TcParams& p) {
  Item it;
  const int blk = t / p.n_chunks;
  it.chunk = t - blk * p.n_chunks;
  const int H = p.heads, D = p.lag;
  if (blk < D) { it.phase = 0; it.head = blk; }
  else {
    const int r = blk - D;
    if (r < 2 * (H - D)) { it.phase = r & 1; it.head = (r & 1) ? (r >> 1) : D + (r >> 1); }
    else { it.phase = 1; it.head = (H - D) + (r - 2 * (H - D)); }
  }
  it.tile0 = it.chunk * p.tiles_per_chunk;
  it.ntiles = min(p.tiles_per_chunk, p.total_tiles - it.tile0);
  return it;
}

// ------------------------------------------------------------------ shared-memory carve-up
constexpr int LSE_SLOTS = 2;
template <int QROWS, int NQ, int STAGES>
struct Smem {
  static constexpr int Q_BYTES = QROWS * HD * 2;
  static constexpr int OFF_Q = 0;
  static constexpr int OFF_K = OFF_Q + NQ * Q_BYTES;
  static constexpr int OFF_LSE = OFF_K + STAGES * KSTAGE_BYTES;   // float[LSE_SLOTS][256]
  static constexpr int OFF_BARS = OFF_LSE + LSE_SLOTS * 256 * 4;
  static constexpr int N_BARS = 2 * STAGES + 2 * NQ + 2 * N_BUFS + 2 * RING + 2 * LSE_SLOTS + 5;
  static constexpr int OFF_SCHED = OFF_BARS + N_BARS * 8;
  static constexpr int OFF_TMEM = OFF_SCHED + RING * 4;
  static constexpr int OFF_REQ = OFF_TMEM + 8;   // {sequence number, head} of the latest merge request
  static constexpr int TOTAL = OFF_REQ + 8;
};

// ------------------------------------------------------------------ epilogue helpers
// one 32-column segment of an S tile: online (max, sum-exp) update of the row this thread owns
__device__ __forceinline__ void s_update(const uint32_t (&v)[32], float sc, float& m, float& z) {
  float g0 = __uint_as_float(v[0]), g1 = __uint_as_float(v[1]);
#pragma unroll
  for (int e = 2; e < 32; e += 2) {
    g0 = fmaxf(g0, __uint_as_float(v[e]));
    g1 = fmaxf(g1, __uint_as_float(v[e + 1]));
  }
  const float m_new = fmaxf(m, fmaxf(g0, g1) * sc);
  float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f;
#pragma unroll
  for (int e = 0; e < 32; e += 4) {
    a0 += fast_exp2(fmaf(__uint_as_float(v[e + 0]), sc, -m_new));
    a1 += fast_exp2(fmaf(__uint_as_float(v[e + 1]), sc, -m_new));
    a2 += fast_exp2(fmaf(__uint_as_float(v[e + 2]), sc, -m_new));
    a3 += fast_exp2(fmaf(__uint_as_float(v[e + 3]), sc, -m_new));
  }
  z = z * fast_exp2(m - m_new) + ((a0 + a1) + (a2 + a3));
  m = m_new;
}

// S tile (128 proxy rows x 128 keys): the TMEM loads of segment s+1 are in flight while segment s is reduced
__device__ __forceinline__ void s_tile(uint32_t tbuf, float sc, float& m, float& z) {
  uint32_t va[32], vb[32];
  tmem_ld32(tbuf, va);
  tc_wait_ld(va);
  tmem_ld32(tbuf + 32, vb);
  s_update(va, sc, m, z);
  tc_wait_ld(vb);
  tmem_ld32(tbuf + 64, va);
  s_update(vb, sc, m, z);
  tc_wait_ld(va);
  tmem_ld32(tbuf + 96, vb);
  s_update(va, sc, m, z);
  tc_wait_ld(vb);
  s_update(vb, sc, m, z);
}

// last tile of a head: columns >= valid are keys past L and must not exist (-inf)
__device__ __forceinline__ void s_tile_masked(uint32_t tbuf, float sc, int valid, float& m, float& z) {
  uint32_t v[32];
#pragma unroll 1
  for (int c = 0; c < valid; c += 32) {
    tmem_ld32(tbuf + c, v);
    tc_wait_ld(v);
#pragma unroll
    for (int e = 0; e < 32; ++e)
      if (c + e >= valid) v[e] = 0xFF800000u;
    s_update(v, sc, m, z);
  }
}

__device__ __forceinline__ void c_update(const uint32_t (&v)[32], int n4, float sc, const float* lse, float& a0, float& a1, float& a2, float& a3) {
  const float4* l4 = reinterpret_cast<const float4*>(lse);
#pragma unroll
  for (int e = 0; e < 8; ++e) {
    if (e < n4) {
      const float4 l = l4[e];
      a0 += fast_exp2(fmaf(__uint_as_float(v[4 * e + 0]), sc, -l.x));
      a1 += fast_exp2(fmaf(__uint_as_float(v[4 * e + 1]), sc, -l.y));
      a2 += fast_exp2(fmaf(__uint_as_float(v[4 * e + 2]), sc, -l.z));
      a3 += fast_exp2(fmaf(__uint_as_float(v[4 * e + 3]), sc, -l.w));
    }
  }
}

// C tile: this thread owns one key; sum over the proxy rows (TMEM columns) of exp2(s*sc - lse2[row])
__device__ __forceinline__ float c_tile(uint32_t tbuf, int rows, float sc, const float* lse) {
  float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f;
  const int nseg = rows >> 5;
  uint32_t va[32], vb[32];
  if (nseg > 0) tmem_ld32(tbuf, va);
#pragma unroll 1
  for (int s = 0; s < nseg; s += 2) {
    tc_wait_ld(va);
    if (s + 1 < nseg) tmem_ld32(tbuf + (s + 1) * 32, vb);
    c_update(va, 8, sc, lse + s * 32, a0, a1, a2, a3);
    if (s + 1 < nseg) {
      tc_wait_ld(vb);
      if (s + 2 < nseg) tmem_ld32(tbuf + (s + 2) * 32, va);
      c_update(vb, 8, sc, lse + (s + 1) * 32, a0, a1, a2, a3);
    }
  }
  if (rows & 16) {
    tmem_ld16(tbuf + nseg * 32, va);
    tc_wait_ld(va);
    c_update(va, 4, sc, lse + nseg * 32, a0, a1, a2, a3);
  }
  return (a0 + a1) + (a2 + a3);
}

// ------------------------------------------------------------------ the kernel
template <int QROWS, int NQ, int STAGES>
__global__ void __launch_bounds__(NTHREADS, 1)
nacl_score_tc_kernel(const __grid_constant__ CUtensorMap tmK, const __grid_constant__ CUtensorMap tmQ, const TcParams p) {
  using SM = Smem<QROWS, NQ, STAGES>;
  extern __shared__ __align__(1024) uint8_t smem[];
  const uint32_t sbase = smem_u32(smem);
  if ((sbase & 1023u) != 0) __trap();  // the 128B-swizzled operand tiles need 1024-byte alignment

  const uint32_t bars = sbase + SM::OFF_BARS;
  constexpr int B_KE = STAGES, B_QF = 2 * STAGES, B_QE = B_QF + NQ, B_TF = B_QE + NQ, B_TE = B_TF + N_BUFS, B_SF = B_TE + N_BUFS,
                B_SE = B_SF + RING, B_LF = B_SE + RING, B_LE = B_LF + LSE_SLOTS, B_DN = B_LE + LSE_SLOTS, B_ACK = B_DN + 2, B_CD = B_ACK + 1, B_SD = B_CD + 1;
  static_assert(B_SD + 1 == SM::N_BARS, "barrier count");
  auto k_full = [&](int s) { return bars + 8u * s; };
  auto k_empty = [&](int s) { return bars + 8u * (B_KE + s); };
  auto q_full = [&](int s) { return bars + 8u * (B_QF + s); };
  auto q_empty = [&](int s) { return bars + 8u * (B_QE + s); };
  auto tm_full = [&](int b) { return bars + 8u * (B_TF + b); };
  auto tm_empty = [&](int b) { return bars + 8u * (B_TE + b); };
  auto sc_full = [&](int s) { return bars + 8u * (B_SF + s); };
  auto sc_empty = [&](int s) { return bars + 8u * (B_SE + s); };
  auto lse_full = [&](int s) { return bars + 8u * (B_LF + s); };
  auto lse_empty = [&](int s) { return bars + 8u * (B_LE + s); };
  auto done_bar = [&](int w) { return bars + 8u * (B_DN + w); };
  const uint32_t ack_bar = bars + 8u * B_ACK, comb_done = bars + 8u * B_CD, sig_done = bars + 8u * B_SD;
  const uint32_t req_addr = sbase + SM::OFF_REQ;
  volatile int* req_head = reinterpret_cast<volatile int*>(smem + SM::OFF_REQ + 4);
  volatile int* sched = reinterpret_cast<volatile int*>(smem + SM::OFF_SCHED);
  volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(smem + SM::OFF_TMEM);
  float* lse_s = reinterpret_cast<float*>(smem + SM::OFF_LSE);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  TR_DECL

  if (threadIdx.x == 0) {
    for (int s = 0; s < STAGES; ++s) { mbar_init(k_full(s), 1); mbar_init(k_empty(s), p.rows > 128 ? 2 : 1); }  // issuers that read a stage
    for (int s = 0; s < NQ; ++s) { mbar_init(q_full(s), 1); mbar_init(q_empty(s), 2); }
    for (int b = 0; b < N_BUFS; ++b) { mbar_init(tm_full(b), 1); mbar_init(tm_empty(b), 4); }
    for (int s = 0; s < RING; ++s) { mbar_init(sc_full(s), 1); mbar_init(sc_empty(s), 3 + N_EPI_WARPS); }
    for (int s = 0; s < LSE_SLOTS; ++s) { mbar_init(lse_full(s), 1); mbar_init(lse_empty(s), N_EPI_WARPS); }
    mbar_init(done_bar(0), 4); mbar_init(done_bar(1), 4); mbar_init(ack_bar, 1);
    mbar_init(comb_done, N_EPI_WARPS); mbar_init(sig_done, 1);
    *reinterpret_cast<volatile uint32_t*>(smem + SM::OFF_REQ) = 0;
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == W_MMA) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(sbase + SM::OFF_TMEM), "r"(TMEM_COLS) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  if (warp == W_TMA) {
    // ================================================================ ticket + TMA producer
    if (lane == 0) {
      int stage = 0;
      uint32_t kphase = 0;
      int qrun = 0, prev_head = -1;
      for (int n = 0;; ++n) {
        const int slot = n % RING;
        TRW(0, mbar_wait(sc_empty(slot), ((n / RING) & 1) ^ 1));
        int t;
        TRW(1, t = atomicAdd(p.ticket, 1));
        if (t >= p.n_items) t = -1;
        sched[slot] = t;
        mbar_arrive(sc_full(slot));
        if (t < 0) break;
        const Item it = decode_item(t, p);
        if (it.head != prev_head) {
          const int qb = qrun % NQ;
          TRW(2, mbar_wait(q_empty(qb), ((qrun / NQ) & 1) ^ 1));
          mbar_expect_tx(q_full(qb), SM::Q_BYTES);
          const uint32_t qdst = sbase + SM::OFF_Q + qb * SM::Q_BYTES;
          tma_load_2d(qdst, &tmQ, 0, it.head * p.rows, q_full(qb));
          tma_load_2d(qdst + QROWS * 128, &tmQ, 64, it.head * p.rows, q_full(qb));
          ++qrun;
          prev_head = it.head;
        }
        for (int i = 0; i < it.ntiles; ++i) {
          TRW(3, mbar_wait(k_empty(stage), kphase ^ 1));
          mbar_expect_tx(k_full(stage), KSTAGE_BYTES);
          const uint32_t kdst = sbase + SM::OFF_K + stage * KSTAGE_BYTES;
          const int j0 = (it.tile0 + i) * TILE;
          tma_load_3d(kdst, &tmK, 0, j0, it.head, k_full(stage));
          tma_load_3d(kdst + BOX_BYTES, &tmK, 64, j0, it.head, k_full(stage));
          if (++stage == STAGES) { stage = 0; kphase ^= 1; }
        }
      }
    }
    __syncwarp();
  } else if (warp == W_MMA || warp == W_MMA + 1) {
    // ================================================================ tcgen05.mma issuer of epilogue warpgroup w
    if (lane == 0) {
      const int w = warp - W_MMA;
      int stage = 0;
      uint32_t kphase = 0;
      int qrun = 0, prev_head = -1;
      uint32_t tcount = 0;
      const uint32_t idesc_s = umma_idesc(128, TILE);
      const bool modeB = p.rows > 128;
      const uint32_t idesc_c = umma_idesc(128, modeB ? min(128, p.rows - 128 * w) : p.rows);
      uint32_t qsrc = 0;
      for (int n = 0;; ++n) {
        const int slot = n % RING;
        TRW(0, mbar_wait(sc_full(slot), (n / RING) & 1));
        const int t = sched[slot];
        mbar_arrive(sc_empty(slot));
        if (t < 0) break;
        const Item it = decode_item(t, p);
        if (it.head != prev_head) {
          if (prev_head >= 0) tc_commit(q_empty((qrun - 1) % NQ));  // every MMA that read the old Q has completed
          const int qb = qrun % NQ;
          TRW(2, mbar_wait(q_full(qb), (qrun / NQ) & 1));
          qsrc = sbase + SM::OFF_Q + qb * SM::Q_BYTES;
          ++qrun;
          prev_head = it.head;
        }
        for (int i = 0; i < it.ntiles; ++i) {
          // rows <= 128: the tile goes to warpgroup (tcount & 1), all proxy rows.
          // rows  > 128: the tile goes to both warpgroups, warpgroup w takes proxy rows [128w, 128w+128).
          if (modeB || (int)(tcount & 1) == w) {
            const uint32_t buf = 2 * w + (modeB ? (tcount & 1) : ((tcount >> 1) & 1));
            const uint32_t par = (modeB ? (tcount >> 1) : (tcount >> 2)) & 1;
            TRW(3, mbar_wait(k_full(stage), kphase));
            TRW(4, mbar_wait(tm_empty(buf), par ^ 1));
            tc_fence_after();
            const uint32_t ksrc = sbase + SM::OFF_K + stage * KSTAGE_BYTES;
            const uint32_t dcol = tmem_base + buf * BUF_COLS;
            const uint32_t qrow = modeB ? w * BOX_BYTES : 0;  // 128 rows x 128 B further down in each Q box
            if (it.phase == 0) {
#pragma unroll
              for (int k = 0; k < 8; ++k) {
                const uint32_t ko = (k >> 2) * BOX_BYTES + (k & 3) * 32;
                const uint32_t qo = (k >> 2) * (QROWS * 128) + (k & 3) * 32 + qrow;
                tc_mma(dcol, umma_desc(qsrc + qo), umma_desc(ksrc + ko), idesc_s, k > 0);
              }
            } else {
#pragma unroll
              for (int k = 0; k < 8; ++k) {
                const uint32_t ko = (k >> 2) * BOX_BYTES + (k & 3) * 32;
                const uint32_t qo = (k >> 2) * (QROWS * 128) + (k & 3) * 32 + qrow;
                tc_mma(dcol, umma_desc(ksrc + ko), umma_desc(qsrc + qo), idesc_c, k > 0);
              }
            }
            tc_commit(tm_full(buf));    // the accumulator buffer is complete
            tc_commit(k_empty(stage));  // this issuer's reads of the stage are done once these MMAs complete
          }
          ++tcount;
          if (++stage == STAGES) { stage = 0; kphase ^= 1; }
        }
      }
    }
    __syncwarp();
  } else if (warp == W_AUX) {
    // ================================================================ helper warp, items in ticket order:
    //   C item: acquire the head's lse flag and stage lse into the shared-memory ring for the epilogue;
    //   S item: once both warpgroups have written their partials, count the chunk; the CTA that counts the last chunk
    //           of a head has its epilogue warps merge the partials, then publishes the head's lse.
    // (One warp serves both: the epilogue is in order too, so an S item cannot finish before the C item ahead of it.)
    int ks = 0, kc = 0;
    uint32_t req_seq = 0;
    for (int n = 0;; ++n) {
      const int slot = n % RING;
      TRW(0, mbar_wait(sc_full(slot), (n / RING) & 1));
      const int t = sched[slot];
      __syncwarp();
      if (lane == 0) mbar_arrive(sc_empty(slot));
      if (t < 0) break;
      const Item it = decode_item(t, p);
      if (it.phase != 0) {
        const int ls = kc % LSE_SLOTS;
        TRW(5, mbar_wait(lse_empty(ls), ((kc / LSE_SLOTS) & 1) ^ 1));
        const long long tf_ = clock64();
        if (lane == 0) {
          uint32_t spins = 0;
          while (ld_acquire(&p.flag[it.head]) == 0) {
            __nanosleep(64);
            if (++spins > (SPIN_LIMIT >> 2)) __trap();
          }
        }
        __syncwarp();
#ifdef NACL_TC_TRACE
        tr_[6] += clock64() - tf_;
#else
        (void)tf_;
#endif
        for (int r = lane; r < p.rows; r += 32) lse_s[ls * 256 + r] = __ldcg(&p.lse2[(size_t)it.head * p.rows + r]);
        __syncwarp();
        if (lane == 0) mbar_arrive(lse_full(ls));
        ++kc;
        continue;
      }
      TRW(7, mbar_wait(done_bar(0), ks & 1); mbar_wait(done_bar(1), ks & 1));
      __syncwarp();
      int last = 0;
      const long long ta_ = clock64();
      if (lane == 0) {
        mbar_arrive(ack_bar);
        __threadfence();  // the warpgroups' partials (ordered before us by the mbarriers) become visible device-wide
        last = (atomicAdd(&p.cnt[it.head], 1) == p.n_chunks - 1) ? 1 : 0;
      }
      last = __shfl_sync(0xffffffffu, last, 0);
#ifdef NACL_TC_TRACE
      tr_[8] += clock64() - ta_;
      const long long tc_ = clock64();
#else
      (void)ta_;
#endif
      if (last) {
        // every chunk of the head is in: the 8 epilogue warps of this CTA merge 32 proxy rows each
        // (they poll the request word at every wait), then the head's lse is published
        if (lane == 0) {
          __threadfence();
          *req_head = it.head;
          sts_release(req_addr, ++req_seq);
        }
        req_seq = __shfl_sync(0xffffffffu, req_seq, 0);
        mbar_wait(comb_done, (req_seq - 1) & 1);
        __syncwarp();
        if (lane == 0) {
          __threadfence();
          st_release(&p.flag[it.head], 1);
        }
#ifdef NACL_TC_TRACE
        tr_[9] += clock64() - tc_;
#endif
      }
      ++ks;
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(sig_done);
  } else {
    // ================================================================ epilogue warpgroups (independent of each other)
    const int wg = warp >> 2, quarter = warp & 3;
    const int lrow = quarter * 32 + lane;             // TMEM lane owned by this thread
    const uint32_t tbase = tmem_base + ((uint32_t)(quarter * 32) << 16);
    const bool modeB = p.rows > 128;
    const int row0 = modeB ? 128 * wg : 0;            // first proxy row this warpgroup is responsible for
    const int nrows_w = min(128, p.rows - row0);      // ... and how many
    const float sc = p.scale_log2;
    const bool live = nrows_w > quarter * 32;         // S items: does this warp own a live proxy row?
    uint32_t ecount = 0;  // tiles seen so far (all items), same sequence as the MMA warp's tcount
    int ks = 0, kc = 0;
    uint32_t seen = 0;    // merge requests served by this warp
    // Every wait of an epilogue warp also serves merge requests of this CTA's signal warp, so a request is
    // answered within one tile and can never deadlock against a wait for another head's lse.
    auto serve = [&]() {
      uint32_t seq = lane == 0 ? lds_acquire(req_addr) : 0u;
      seq = __shfl_sync(0xffffffffu, seq, 0);
      if (seq == seen) return;
      seen = seq;
#ifdef NACL_TC_TRACE
      const long long tm_ = clock64();
#endif
      const int head = *req_head;
      const int r = warp * 32 + lane;
      if (r < p.rows) {
        const size_t row = (size_t)head * p.rows + r;
        const int np = p.n_chunks * p.n_slots;  // partials per row
        const float l2 = merge_row(p.part + (size_t)head * np * p.rows + r, np, (size_t)p.rows);
        __stcg(&p.lse2[row], l2);
        if (p.lse_out) p.lse_out[row] = l2 * 0.69314718055994530942f;
      }
#ifdef NACL_TC_TRACE
      tr_[6] += clock64() - tm_;
      const long long tq_ = clock64();
#endif
      __threadfence();
      __syncwarp();
#ifdef NACL_TC_TRACE
      tr_[7] += clock64() - tq_;
      tr_[8] += 1;
#endif
      if (lane == 0) mbar_arrive(comb_done);
    };
    auto ewait = [&](uint32_t bar, uint32_t parity) {
      serve();  // also when the barrier is already complete: a busy epilogue may not block for a long time
      uint32_t spins = 0;
      while (!__all_sync(0xffffffffu, mbar_try_wait(bar, parity))) {
        serve();
        if (++spins > SPIN_LIMIT) __trap();
      }
    };
    for (int n = 0;; ++n) {
      const int slot = n % RING;
      TRW(0, ewait(sc_full(slot), (n / RING) & 1));
      const int t = sched[slot];
      __syncwarp();
      if (lane == 0) mbar_arrive(sc_empty(slot));
      if (t < 0) break;
      const Item it = decode_item(t, p);
      if (it.phase == 0) {
        // ---------------- S item: running (max, sum-exp) of rows lrow (and 128 + lrow) over this warpgroup's tiles
        float m0 = -INFINITY, z0 = 0.f;
        for (int i = 0; i < it.ntiles; ++i) {
          const uint32_t g = ecount + i;
          if (!modeB && (int)(g & 1) != wg) continue;
          const uint32_t buf = 2 * wg + (modeB ? (g & 1) : ((g >> 1) & 1));
          TRW(10, ewait(tm_full(buf), (modeB ? (g >> 1) : (g >> 2)) & 1));
          tc_fence_after();
          const long long ts_ = clock64();
          const int valid = p.L - (it.tile0 + i) * TILE;
          if (live) {
            if (valid >= TILE) s_tile(tbase + buf * BUF_COLS, sc, m0, z0);
            else s_tile_masked(tbase + buf * BUF_COLS, sc, valid, m0, z0);
          }
          tc_fence_before();
          __syncwarp();
#ifdef NACL_TC_TRACE
          tr_[11] += clock64() - ts_;
#else
          (void)ts_;
#endif
          if (lane == 0) mbar_arrive(tm_empty(buf));
        }
        ecount += it.ntiles;
        // this warpgroup's partial of the chunk; (-inf, 0) when it saw no tile
        if (lrow < nrows_w)
          __stcg(&p.part[(((size_t)it.head * p.n_chunks + it.chunk) * p.n_slots + (modeB ? 0 : wg)) * p.rows + row0 + lrow], make_float2(m0, z0));
        if (ks > 0) TRW(12, ewait(ack_bar, (ks - 1) & 1));  // the signal warp has consumed our previous arrival
        __syncwarp();
        if (lane == 0) mbar_arrive(done_bar(wg));
        ++ks;
      } else {
        // ---------------- C item: column sums with the lse the loader warp staged
        const int ls = kc % LSE_SLOTS;
        TRW(5, ewait(lse_full(ls), (kc / LSE_SLOTS) & 1));
        const float* lse = lse_s + ls * 256;
        for (int i = 0; i < it.ntiles; ++i) {
          const uint32_t g = ecount + i;
          if (!modeB && (int)(g & 1) != wg) continue;
          const uint32_t buf = 2 * wg + (modeB ? (g & 1) : ((g >> 1) & 1));
          TRW(13, ewait(tm_full(buf), (modeB ? (g >> 1) : (g >> 2)) & 1));
          tc_fence_after();
          float r;
          TRW(14, r = c_tile(tbase + buf * BUF_COLS, nrows_w, sc, lse + row0));
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(tm_empty(buf));
          const int j = (it.tile0 + i) * TILE + lrow;
          if (j < p.L) {
            const size_t o = (size_t)it.head * p.L + j;
            if (modeB) {
              // two addends per element onto a zeroed word: a + b == b + a bit for bit, whichever arrives first
              atomicAdd(&p.imp[o], r);
              if (p.imp_out) atomicAdd(&p.imp_out[o], r);
            } else {
              p.imp[o] = r;
              if (p.imp_out) p.imp_out[o] = r;
            }
          }
        }
        ecount += it.ntiles;
        __syncwarp();
        if (lane == 0) mbar_arrive(lse_empty(ls));
        ++kc;
      }
    }
    ewait(sig_done, 0);  // keep serving until this CTA's signal warp has nothing left to ask
  }

  TR_FLUSH()
  tc_fence_before();
  __syncthreads();
  if (warp == W_MMA) {
    tc_fence_after();
    __syncwarp();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(TMEM_COLS) : "memory");
  }
}

// ------------------------------------------------------------------ host side
using EncodeTiledFn = CUresult (*)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                   const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                   CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_tiled_fn() {
  static EncodeTiledFn fn = [] {
    void* f = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess)
      f = nullptr;
    return reinterpret_cast<EncodeTiledFn>(f);
  }();
  return fn;
}

int sm_count() {
  static int n = [] {
    int dev = 0, v = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || v <= 0)
      v = kNumSMs;
    return v;
  }();
  return n;
}

template <int QROWS, int NQ, int STAGES>
cudaError_t launch_cfg(const CUtensorMap& tmK, const CUtensorMap& tmQ, const TcParams& p, cudaStream_t st) {
  using SM = Smem<QROWS, NQ, STAGES>;
  static_assert(SM::TOTAL <= 227 * 1024, "shared memory budget");
  auto kern = nacl_score_tc_kernel<QROWS, NQ, STAGES>;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, SM::TOTAL);
  if (e != cudaSuccess) return e;
  const int grid = p.n_items < sm_count() ? p.n_items : sm_count();
  kern<<<grid, NTHREADS, SM::TOTAL, st>>>(tmK, tmQ, p);
  return cudaGetLastError();
}

}  // namespace

bool score_tc_supported(const Shape& s) {
  return s.dtype == NACL_DTYPE_BF16 && s.d == HD && s.rows % 16 == 0 && s.rows >= 16 && s.rows <= 256;
}

int score_tc_launch_count(const Shape&) { return 1; }

cudaError_t launch_score_tc(const Shape& s, const void* K, const void* Q, const SplitPlan& sp, const Workspace& ws,
                            float* imp_out, float* lse_out, cudaStream_t st) {
  EncodeTiledFn enc = encode_tiled_fn();
  if (!enc) return cudaErrorNotSupported;  // no silent fallback: the caller reports NACL_ERR_CUDA
  const int heads = s.batch * s.Hkv;
  const int qrows = s.rows <= 128 ? 128 : 256;

  alignas(64) CUtensorMap tmK, tmQ;
  {
    const cuuint64_t dims[3] = {(cuuint64_t)HD, (cuuint64_t)s.L, (cuuint64_t)heads};
    const cuuint64_t strides[2] = {(cuuint64_t)HD * 2, (cuuint64_t)s.L * HD * 2};
    const cuuint32_t box[3] = {64, (cuuint32_t)TILE, 1};
    const cuuint32_t es[3] = {1, 1, 1};
    if (enc(&tmK, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(K), dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
            CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return cudaErrorInvalidValue;
  }
  {
    const cuuint64_t dims[2] = {(cuuint64_t)HD, (cuuint64_t)heads * s.rows};
    const cuuint64_t strides[1] = {(cuuint64_t)HD * 2};
    const cuuint32_t box[2] = {64, (cuuint32_t)qrows};
    const cuuint32_t es[2] = {1, 1};
    if (enc(&tmQ, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(Q), dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
            CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return cudaErrorInvalidValue;
  }

  TcParams p;
  p.L = s.L; p.rows = s.rows; p.n_halves = (s.rows + 127) / 128;
  p.n_chunks = sp.n_chunks; p.tiles_per_chunk = sp.chunk / TILE; p.total_tiles = (s.L + TILE - 1) / TILE;
  p.heads = heads;
  p.n_slots = s.rows <= 128 ? 2 : 1;
  // lag in heads between the first and the second read of a head's K: a few heads, at most ~48 MB of K in between
  const size_t head_bytes = (size_t)s.L * HD * 2;
  int lag = (int)((size_t)64 * 1024 * 1024 / head_bytes);
  lag = lag < 1 ? 1 : (lag > 8 ? 8 : lag);
  p.lag = lag < heads ? lag : heads;
  p.n_items = 2 * heads * sp.n_chunks;
  p.scale_log2 = 1.4426950408889634f / sqrtf((float)s.d);
  p.ticket = ws.sync; p.cnt = ws.sync + 16; p.flag = ws.sync + 16 + heads;
  p.part = ws.part; p.lse2 = ws.lse; p.lse_out = lse_out; p.imp = ws.imp; p.imp_out = imp_out;

  cudaError_t e = cudaMemsetAsync(ws.sync, 0, (size_t)(16 + 2 * heads) * sizeof(int), st);
  if (e != cudaSuccess) return e;
  if (s.rows > 128) {  // each importance is the sum of two warpgroup partials added onto zero (see the C items)
    if ((e = cudaMemsetAsync(ws.imp, 0, (size_t)heads * s.L * sizeof(float), st)) != cudaSuccess) return e;
    if (imp_out && (e = cudaMemsetAsync(imp_out, 0, (size_t)heads * s.L * sizeof(float), st)) != cudaSuccess) return e;
  }
  StageScope sc(ST_FUSED, st);
  if (qrows == 128) return launch_cfg<128, 2, 5>(tmK, tmQ, p, st);
  return launch_cfg<256, 2, 3>(tmK, tmQ, p, st);
}


}  // namespace nacl

#ifdef NACL_TC_TRACE
// diagnostics build only: per-warp wait/compute cycle counters of the last launch
extern "C" __attribute__((visibility("default"))) int nacl_debug_trace_read(long long* host, size_t bytes) {
  return (int)cudaMemcpyFromSymbol(host, nacl::g_trace, bytes < sizeof(nacl::g_trace) ? bytes : sizeof(nacl::g_trace));
}
#endif
