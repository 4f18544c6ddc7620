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
constexpr int NTHREADS = EPI_THREADS + 64;
constexpr int RING = 4;                        // ticket ring slots
constexpr int TMEM_COLS = 512;
constexpr int BUF_COLS = 256;                  // TMEM columns per accumulator buffer
constexpr uint32_t SPIN_LIMIT = 1u << 24;      // watchdog: a wait that long is a bug -> trap (loud failure)

struct TcParams {
  int L, rows, n_halves, n_chunks, tiles_per_chunk, total_tiles;
  int heads, lag, n_items;
  float scale_log2;   // log2(e) / sqrt(d)
  int* ticket;        // [1]
  int* cnt;           // [heads]  finished S items per head
  int* flag;          // [heads]  1 once lse of the head is published
  float2* part;       // [heads*rows, n_chunks]  (m, z) in the log2 domain
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
__device__ __forceinline__ void tc_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

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
__device__ __forceinline__ void epi_bar() { asm volatile("bar.sync 1, %0;" ::"n"(EPI_THREADS) : "memory"); }

__device__ __forceinline__ int ld_acquire(const int* p) {
  int v;
  asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_release(int* p, int v) {
  asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// K-major operand tile, 128-byte swizzle, rows of 128 B, 8-row groups 1024 B apart (sm_100 descriptor v1)
__device__ __forceinline__ uint64_t umma_desc(uint32_t smem_addr) {
  return (uint64_t)((smem_addr >> 4) & 0x3FFFu) | (1ull << 16) | (64ull << 32) | (1ull << 46) | (2ull << 61);
}
// kind::f16 instruction descriptor: D fp32, A/B bf16, both K-major
__device__ __forceinline__ uint32_t umma_idesc(int M, int N) {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}

// merge two (max, sum-exp) partials in the log2 domain; (-inf, 0) is the identity
__device__ __forceinline__ void merge2(float& m, float& z, float m2, float z2) {
  const float mn = fmaxf(m, m2);
  if (mn == -INFINITY) { m = mn; z = 0.f; return; }
  z = z * exp2f(m - mn) + z2 * exp2f(m2 - mn);
  m = mn;
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
template <int QROWS, int NQ, int STAGES>
struct Smem {
  static constexpr int Q_BYTES = QROWS * HD * 2;
  static constexpr int OFF_Q = 0;
  static constexpr int OFF_K = OFF_Q + NQ * Q_BYTES;
  static constexpr int OFF_AUX = OFF_K + STAGES * KSTAGE_BYTES;
  // aux: barriers, ticket ring, tmem base, reduction scratch
  static constexpr int N_BARS = 2 * STAGES + 2 * NQ + 4 + 2 * RING;
  static constexpr int OFF_BARS = OFF_AUX;
  static constexpr int OFF_SCHED = OFF_BARS + N_BARS * 8;
  static constexpr int OFF_TMEM = OFF_SCHED + RING * 4;
  static constexpr int OFF_LAST = OFF_TMEM + 4;
  static constexpr int OFF_RED = (OFF_LAST + 4 + 15) / 16 * 16;  // float2[256]
  static constexpr int OFF_LSE = OFF_RED + 256 * 8;              // float[256]
  static constexpr int TOTAL = OFF_LSE + 256 * 4;
};

// ------------------------------------------------------------------ the kernel
template <int QROWS, int NQ, int STAGES>
__global__ void __launch_bounds__(NTHREADS, 1)
nacl_score_tc_kernel(const __grid_constant__ CUtensorMap tmK, const __grid_constant__ CUtensorMap tmQ, const TcParams p) {
  using SM = Smem<QROWS, NQ, STAGES>;
  extern __shared__ __align__(1024) uint8_t smem[];
  const uint32_t sbase = smem_u32(smem);
  if ((sbase & 1023u) != 0) __trap();  // the 128B-swizzled operand tiles need 1024-byte alignment

  const uint32_t bars = sbase + SM::OFF_BARS;
  auto k_full = [&](int s) { return bars + 8u * s; };
  auto k_empty = [&](int s) { return bars + 8u * (STAGES + s); };
  auto q_full = [&](int s) { return bars + 8u * (2 * STAGES + s); };
  auto q_empty = [&](int s) { return bars + 8u * (2 * STAGES + NQ + s); };
  auto tm_full = [&](int b) { return bars + 8u * (2 * STAGES + 2 * NQ + b); };
  auto tm_empty = [&](int b) { return bars + 8u * (2 * STAGES + 2 * NQ + 2 + b); };
  auto sc_full = [&](int s) { return bars + 8u * (2 * STAGES + 2 * NQ + 4 + s); };
  auto sc_empty = [&](int s) { return bars + 8u * (2 * STAGES + 2 * NQ + 4 + RING + s); };
  volatile int* sched = reinterpret_cast<volatile int*>(smem + SM::OFF_SCHED);
  volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(smem + SM::OFF_TMEM);
  volatile int* last_flag = reinterpret_cast<volatile int*>(smem + SM::OFF_LAST);
  float2* red = reinterpret_cast<float2*>(smem + SM::OFF_RED);
  float* lse_s = reinterpret_cast<float*>(smem + SM::OFF_LSE);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (threadIdx.x == 0) {
    for (int s = 0; s < STAGES; ++s) { mbar_init(k_full(s), 1); mbar_init(k_empty(s), 1); }
    for (int s = 0; s < NQ; ++s) { mbar_init(q_full(s), 1); mbar_init(q_empty(s), 1); }
    for (int b = 0; b < 2; ++b) { mbar_init(tm_full(b), 1); mbar_init(tm_empty(b), 4); }
    for (int s = 0; s < RING; ++s) { mbar_init(sc_full(s), 1); mbar_init(sc_empty(s), 1 + N_EPI_WARPS); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 9) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(sbase + SM::OFF_TMEM), "r"(TMEM_COLS) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  if (warp == 8) {
    // ================================================================ ticket + TMA producer
    if (lane == 0) {
      int stage = 0;
      uint32_t kphase = 0;
      int qrun = 0, prev_head = -1;
      for (int n = 0;; ++n) {
        const int slot = n % RING;
        mbar_wait(sc_empty(slot), ((n / RING) & 1) ^ 1);
        int t = atomicAdd(p.ticket, 1);
        if (t >= p.n_items) t = -1;
        sched[slot] = t;
        mbar_arrive(sc_full(slot));
        if (t < 0) break;
        const Item it = decode_item(t, p);
        if (it.head != prev_head) {
          const int qb = qrun % NQ;
          mbar_wait(q_empty(qb), ((qrun / NQ) & 1) ^ 1);
          mbar_expect_tx(q_full(qb), SM::Q_BYTES);
          const uint32_t qdst = sbase + SM::OFF_Q + qb * SM::Q_BYTES;
          tma_load_2d(qdst, &tmQ, 0, it.head * p.rows, q_full(qb));
          tma_load_2d(qdst + QROWS * 128, &tmQ, 64, it.head * p.rows, q_full(qb));
          ++qrun;
          prev_head = it.head;
        }
        for (int i = 0; i < it.ntiles; ++i) {
          mbar_wait(k_empty(stage), kphase ^ 1);
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
  } else if (warp == 9) {
    // ================================================================ tcgen05.mma issuer
    if (lane == 0) {
      int stage = 0;
      uint32_t kphase = 0;
      int qrun = 0, prev_head = -1;
      uint32_t tcount = 0;
      const uint32_t idesc_s = umma_idesc(128, TILE);
      const uint32_t idesc_c = umma_idesc(128, p.rows);
      uint32_t qsrc = 0;
      for (int n = 0;; ++n) {
        const int slot = n % RING;
        mbar_wait(sc_full(slot), (n / RING) & 1);
        const int t = sched[slot];
        mbar_arrive(sc_empty(slot));
        if (t < 0) break;
        const Item it = decode_item(t, p);
        if (it.head != prev_head) {
          if (prev_head >= 0) tc_commit(q_empty((qrun - 1) % NQ));  // every MMA that read the old Q has completed
          const int qb = qrun % NQ;
          mbar_wait(q_full(qb), (qrun / NQ) & 1);
          qsrc = sbase + SM::OFF_Q + qb * SM::Q_BYTES;
          ++qrun;
          prev_head = it.head;
        }
        for (int i = 0; i < it.ntiles; ++i) {
          const uint32_t b = tcount & 1;
          mbar_wait(tm_empty(b), ((tcount >> 1) & 1) ^ 1);
          mbar_wait(k_full(stage), kphase);
          tc_fence_after();
          const uint32_t ksrc = sbase + SM::OFF_K + stage * KSTAGE_BYTES;
          const uint32_t dcol = tmem_base + b * BUF_COLS;
          if (it.phase == 0) {
            for (int h = 0; h < p.n_halves; ++h) {
#pragma unroll
              for (int k = 0; k < 8; ++k) {
                const uint32_t ko = (k >> 2) * BOX_BYTES + (k & 3) * 32;
                const uint32_t qo = (k >> 2) * (QROWS * 128) + (k & 3) * 32 + h * BOX_BYTES;
                tc_mma(dcol + h * TILE, umma_desc(qsrc + qo), umma_desc(ksrc + ko), idesc_s, k > 0);
              }
            }
          } else {
#pragma unroll
            for (int k = 0; k < 8; ++k) {
              const uint32_t ko = (k >> 2) * BOX_BYTES + (k & 3) * 32;
              const uint32_t qo = (k >> 2) * (QROWS * 128) + (k & 3) * 32;
              tc_mma(dcol, umma_desc(ksrc + ko), umma_desc(qsrc + qo), idesc_c, k > 0);
            }
          }
          tc_commit(k_empty(stage));  // the stage may be refilled once these MMAs have read it
          tc_commit(tm_full(b));      // the accumulator buffer is complete
          ++tcount;
          if (++stage == STAGES) { stage = 0; kphase ^= 1; }
        }
      }
    }
    __syncwarp();
  } else {
    // ================================================================ epilogue warpgroups
    const int wg = warp >> 2, quarter = warp & 3;
    const int tid = threadIdx.x;                      // 0..255
    const int lrow = quarter * 32 + lane;             // TMEM lane owned by this thread
    const uint32_t tbuf = tmem_base + ((uint32_t)(quarter * 32) << 16) + wg * BUF_COLS;
    const float sc = p.scale_log2;
    uint32_t ecount = 0;  // tiles seen so far (all items), same sequence as the MMA warp's tcount
    for (int n = 0;; ++n) {
      const int slot = n % RING;
      mbar_wait(sc_full(slot), (n / RING) & 1);
      const int t = sched[slot];
      __syncwarp();
      if (lane == 0) mbar_arrive(sc_empty(slot));
      if (t < 0) break;
      const Item it = decode_item(t, p);
      if (it.phase == 0) {
        // ---------------- S item: running (max, sum-exp) of rows lrow (and 128 + lrow)
        float m[2] = {-INFINITY, -INFINITY}, z[2] = {0.f, 0.f};
        for (int i = 0; i < it.ntiles; ++i) {
          const uint32_t g = ecount + i;
          if ((int)(g & 1) != wg) continue;
          mbar_wait(tm_full(wg), (g >> 1) & 1);
          tc_fence_after();
          const int valid = min(TILE, p.L - (it.tile0 + i) * TILE);
          for (int h = 0; h < p.n_halves; ++h) {
            if (h * 128 + quarter * 32 >= p.rows) continue;  // warp-uniform: no live proxy row in this warp
            uint32_t v[32];
#pragma unroll 1
            for (int c = 0; c < 4; ++c) {
              tmem_ld32(tbuf + h * TILE + c * 32, v);
              tc_wait_ld();
              if (valid < TILE) {
#pragma unroll
                for (int e = 0; e < 32; ++e)
                  if (c * 32 + e >= valid) v[e] = 0xFF800000u;  // -inf: keys past L do not exist
              }
              float gmax = __uint_as_float(v[0]);
#pragma unroll
              for (int e = 1; e < 32; ++e) gmax = fmaxf(gmax, __uint_as_float(v[e]));
              const float m_new = fmaxf(m[h], gmax * sc);
              float zz0 = 0.f, zz1 = 0.f;
#pragma unroll
              for (int e = 0; e < 32; e += 2) {
                zz0 += fast_exp2(fmaf(__uint_as_float(v[e]), sc, -m_new));
                zz1 += fast_exp2(fmaf(__uint_as_float(v[e + 1]), sc, -m_new));
              }
              z[h] = z[h] * fast_exp2(m[h] - m_new) + (zz0 + zz1);
              m[h] = m_new;
            }
          }
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(tm_empty(wg));
        }
        ecount += it.ntiles;
        // ---------------- merge the two warpgroups, write the chunk partial, count the chunk
        if (wg == 1) {
          red[lrow] = make_float2(m[0], z[0]);
          red[128 + lrow] = make_float2(m[1], z[1]);
        }
        epi_bar();
        if (wg == 0) {
#pragma unroll
          for (int h = 0; h < 2; ++h) {
            const int r = h * 128 + lrow;
            if (r < p.rows) {
              const float2 o = red[r];
              float mm = m[h], zz = z[h];
              merge2(mm, zz, o.x, o.y);
              __stcg(&p.part[((size_t)it.head * p.rows + r) * p.n_chunks + it.chunk], make_float2(mm, zz));
            }
          }
          __threadfence();
        }
        epi_bar();
        if (tid == 0) *last_flag = (atomicAdd(&p.cnt[it.head], 1) == p.n_chunks - 1) ? 1 : 0;
        epi_bar();
        if (*last_flag) {
          // this CTA finished the last S item of the head: merge the chunks in ascending order
          __threadfence();
          if (tid < p.rows) {
            const size_t row = (size_t)it.head * p.rows + tid;
            float mm = -INFINITY, zz = 0.f;
            for (int c = 0; c < p.n_chunks; ++c) {
              const float2 o = __ldcg(&p.part[row * p.n_chunks + c]);
              merge2(mm, zz, o.x, o.y);
            }
            const float l2 = mm + log2f(zz);
            __stcg(&p.lse2[row], l2);
            if (p.lse_out) p.lse_out[row] = l2 * 0.69314718055994530942f;
          }
          __threadfence();
          epi_bar();
          if (tid == 0) st_release(&p.flag[it.head], 1);
        }
      } else {
        // ---------------- C item: wait for lse of the head, then column sums
        if (tid == 0) {
          uint32_t spins = 0;
          while (ld_acquire(&p.flag[it.head]) == 0) {
            __nanosleep(100);
            if (++spins > (SPIN_LIMIT >> 2)) __trap();
          }
        }
        epi_bar();  // also: every thread is done with lse_s of the previous C item
        if (tid < p.rows) lse_s[tid] = __ldcg(&p.lse2[(size_t)it.head * p.rows + tid]);
        epi_bar();
        for (int i = 0; i < it.ntiles; ++i) {
          const uint32_t g = ecount + i;
          if ((int)(g & 1) != wg) continue;
          mbar_wait(tm_full(wg), (g >> 1) & 1);
          tc_fence_after();
          float acc0 = 0.f, acc1 = 0.f;
          uint32_t v[32];
          int c0 = 0;
#pragma unroll 1
          for (; c0 + 32 <= p.rows; c0 += 32) {
            tmem_ld32(tbuf + c0, v);
            tc_wait_ld();
            const float4* l4 = reinterpret_cast<const float4*>(lse_s + c0);
#pragma unroll
            for (int e = 0; e < 8; ++e) {
              const float4 l = l4[e];
              acc0 += fast_exp2(fmaf(__uint_as_float(v[4 * e + 0]), sc, -l.x));
              acc1 += fast_exp2(fmaf(__uint_as_float(v[4 * e + 1]), sc, -l.y));
              acc0 += fast_exp2(fmaf(__uint_as_float(v[4 * e + 2]), sc, -l.z));
              acc1 += fast_exp2(fmaf(__uint_as_float(v[4 * e + 3]), sc, -l.w));
            }
          }
          if (c0 < p.rows) {  // rows % 32 == 16
            tmem_ld16(tbuf + c0, v);
            tc_wait_ld();
            const float4* l4 = reinterpret_cast<const float4*>(lse_s + c0);
#pragma unroll
            for (int e = 0; e < 4; ++e) {
              const float4 l = l4[e];
              acc0 += fast_exp2(fmaf(__uint_as_float(v[4 * e + 0]), sc, -l.x));
              acc1 += fast_exp2(fmaf(__uint_as_float(v[4 * e + 1]), sc, -l.y));
              acc0 += fast_exp2(fmaf(__uint_as_float(v[4 * e + 2]), sc, -l.z));
              acc1 += fast_exp2(fmaf(__uint_as_float(v[4 * e + 3]), sc, -l.w));
            }
          }
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(tm_empty(wg));
          const int j = (it.tile0 + i) * TILE + lrow;
          if (j < p.L) {
            const float r = acc0 + acc1;
            const size_t o = (size_t)it.head * p.L + j;
            p.imp[o] = r;
            if (p.imp_out) p.imp_out[o] = r;
          }
        }
        ecount += it.ntiles;
      }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 9) {
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
  // lag in heads between the first and the second read of a head's K: a few heads, at most ~48 MB of K in between
  const size_t head_bytes = (size_t)s.L * HD * 2;
  int lag = (int)((size_t)48 * 1024 * 1024 / head_bytes);
  lag = lag < 1 ? 1 : (lag > 4 ? 4 : lag);
  p.lag = lag < heads ? lag : heads;
  p.n_items = 2 * heads * sp.n_chunks;
  p.scale_log2 = 1.4426950408889634f / sqrtf((float)s.d);
  p.ticket = ws.sync; p.cnt = ws.sync + 16; p.flag = ws.sync + 16 + heads;
  p.part = ws.part; p.lse2 = ws.lse; p.lse_out = lse_out; p.imp = ws.imp; p.imp_out = imp_out;

  cudaError_t e = cudaMemsetAsync(ws.sync, 0, (size_t)(16 + 2 * heads) * sizeof(int), st);
  if (e != cudaSuccess) return e;
  StageScope sc(ST_FUSED, st);
  if (qrows == 128) return launch_cfg<128, 2, 4>(tmK, tmQ, p, st);
  return launch_cfg<256, 1, 4>(tmK, tmQ, p, st);
}

}  // namespace nacl
