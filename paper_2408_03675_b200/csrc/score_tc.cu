// score_tc.cu -- tensor-core scoring path: steps a1-a3 of SURVEY.md section 8 as a persistent,
// warp-specialised sm_100a kernel (tcgen05.mma + TMEM accumulators + TMA-staged tiles).  Both sweeps
// run in ONE cooperative launch (nacl_evict_ex), or as two plain launches (nacl_evict_batch, where the
// calls of two streams share the GPU; NACL_FLAG_SCORE_TWO_LAUNCHES; sweep C alone when lse_in is given):
//
//   a1  s[i,j] = Q[i,:].K[j,:] / sqrt(d)                      PAPER.md:59, Alg.1
//   a2  lse_i  = log sum_j exp(s[i,j])   (full-length softmax)  PAPER.md:124      -- sweep S
//   a3  imp[j] = sum_{g,i} exp(s[i,j] - lse_i)                  PAPER.md:124, 176-178 -- sweep C
//
// Serves bf16, d == 128, G*P a multiple of 16 (above 256: in blocks of 256 proxy rows), contiguous, strided or paged K.
// Everything else takes score_generic.cu.
//
// Work decomposition.  The logits are never written to memory and the column sum needs the
// complete row normaliser first, so every key tile (128 keys) is scored twice.  The N = heads * T
// key tiles of a call (T = ceil(L/128) per kv head) form one flat sequence that is cut into
// gridDim.x equal contiguous ranges: CTA c owns tiles [N*c/G, N*(c+1)/G) in BOTH sweeps -- no
// tickets and no float atomics; the only inter-CTA wait is the hand-over of a head's partials in the
// one-launch form (a per-head counter).  A range crosses at most a few head boundaries; each
// maximal run of tiles of one head is a segment.  Every K tile load carries the L2 evict_first hint.
//   sweep S: per segment and proxy row a partial (max, sum-exp) is written to part[c + head]
//            (c + head is strictly increasing along the sequence, hence a unique slot);
//   sweep C: the CTA first merges, per segment, the head's partials in ascending slot order into
//            lse (fixed order: deterministic), then walks its range BACKWARDS, so the tiles it read
//            last in sweep S -- still resident in the 126 MB L2 -- are read first.
// No floating-point atomics with more than two addends anywhere: all sums have a fixed order.
//
// Two MMA orientations share the same shared-memory operands (both K-major, 128B swizzle):
//   S tiles:  D[row, key] = Q_half (M=128 proxy rows) x K_tile^T (N=128 keys), one MMA group per
//             128-row half -> a thread owns a proxy row and a range of key columns; its running
//             (max, sum-exp) live in two registers;
//   C tiles:  D[key, row] = K_tile (M=128 keys) x Q^T (N = G*P proxy rows) -> a thread owns a key
//             and a quarter of the proxy rows; the four quarter sums of a key meet in shared memory
//             and a combiner warp adds them in a fixed order (deterministic) and stores imp.
//
// Epilogue arithmetic.  At G*P = 256 the path is bound by TMEM loads + the 16/clk/SM MUFU.EX2 unit + the
// FMA pipe, not by HBM (profiles/): 3 of 8 exponentials are therefore evaluated on the FMA pipe
// (saturating-FMA range reduction + degree-3 minimax polynomial, relative error <= 7.5e-5, against the
// 2e-3 score tolerance of the north star) and all multiply-adds are the packed fma/add.f32x2 forms.
//
// Warp roles (640 threads, 1 CTA per SM): warps 0-15 = epilogue (warp%4 = TMEM lane quarter = SM
// sub-partition, warp/4 = column quarter of the tile, or (tile parity, row half) in the quad scheme),
// warp 16 = TMA producer, warps 17-18 = tcgen05.mma issuers (alternating tiles; 17 also allocates TMEM),
// warp 19 = column-sum combiner in sweep C, publisher of the partials in sweep S of the one-launch form.
#include <cuda.h>

#include "nacl_internal.cuh"

namespace nacl {
namespace {

constexpr int TILE = 128;                      // keys per tile
constexpr int HD = 128;                        // head dim served by this path
constexpr int BOX_BYTES = 128 * 128;           // one TMA box: 128 rows x 64 bf16 (128 B, swizzled)
constexpr int KSTAGE_BYTES = 2 * BOX_BYTES;    // a K tile = two boxes (d 0..63, d 64..127)
constexpr int N_EPI_WARPS = 16;
constexpr int EPI_THREADS = N_EPI_WARPS * 32;
constexpr int W_TMA = 16, W_MMA = 17, W_MMA2 = 18, W_CMB = 19;  // warp roles after the epilogue warps
constexpr int NTHREADS = EPI_THREADS + 4 * 32;
constexpr int TMEM_COLS = 512;
constexpr int N_BUFS = 2;                      // TMEM accumulator buffers (one tile each)
constexpr int BUF_COLS = 256;                  // TMEM columns per accumulator buffer
constexpr int N_CS = 4;                        // shared-memory buffers for the quarter column sums of a C tile
constexpr int MAX_GRID = kNumSMs;              // the partial-statistics workspace is sized for this many CTAs
constexpr uint32_t SPIN_LIMIT = 1u << 26;      // watchdog: a wait that long is a bug -> trap (loud failure)
// which of every 8 element pairs take the FMA-pipe exp2 instead of MUFU.EX2 (bit e&7), per sweep: measured optimum on
// B200 (cfg 4, us per layer): sweep S 74.8 / 71.9 / 75.3 for 2/8, 3/8, 4/8; sweep C 78.2 / 76.2 for 2/8, 3/8
#ifndef NACL_POLY_MASK_S
#define NACL_POLY_MASK_S 0x2Au
#endif
#ifndef NACL_POLY_MASK_C
#define NACL_POLY_MASK_C 0x2Au
#endif

// Optional wait/compute cycle accounting per warp role (diagnostics build only: -DNACL_TC_TRACE).
#ifdef NACL_TC_TRACE
#define TR_N 8
__device__ long long g_trace[2][160][20][TR_N];
__device__ __forceinline__ long long gtimer_ns() { long long t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); return t; }
#define TR_DECL long long tr_[TR_N]; for (int i_ = 0; i_ < TR_N; ++i_) tr_[i_] = 0; const long long tr_start_ = clock64(); const long long tr_ns_ = gtimer_ns();
#define TRW(cat, ...) { const long long t_ = clock64(); __VA_ARGS__; tr_[cat] += clock64() - t_; }
__device__ long long g_tl[2][20][32][8];
#define TL(k) { if (blockIdx.x == 40 && lane == 0 && tl_i_ >= 0 && tl_i_ < 32) g_tl[PH][warp][tl_i_][k] = clock64(); }
#define TL_NEXT() { ++tl_i_; }
#define TL_DECL int tl_i_ = -8;
#define TL2(k) { if (blockIdx.x == 40 && (threadIdx.x & 31) == 0 && tl_i_ >= 0 && tl_i_ < 32) g_tl[0][threadIdx.x >> 5][tl_i_][k] = clock64(); }
#define TR_FLUSH() { tr_[TR_N - 1] = clock64() - tr_start_; tr_[TR_N - 2] = gtimer_ns() - tr_ns_; if (lane == 0 && blockIdx.x < 160) for (int i_ = 0; i_ < TR_N; ++i_) g_trace[PH][blockIdx.x][warp][i_] = tr_[i_]; }
#else
#define TR_DECL
#define TRW(cat, ...) { __VA_ARGS__; }
#define TR_FLUSH()
#define TL(k)
#define TL_NEXT()
#define TL_DECL
#define TL2(k)
#endif

// Optional globaltimer stamps of every CTA (diagnostics build only: -DNACL_TC_STAMPS): kernel entry, TMEM allocated,
// sweep S done, sweep C done.
#ifdef NACL_TC_STAMPS
__device__ long long g_stamps[160][4];
#define GSTAMP(k) { if (threadIdx.x == 0 && blockIdx.x < 160) { long long t_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_)); g_stamps[blockIdx.x][k] = t_; } }
#else
#define GSTAMP(k)
#endif

struct TcParams {
  int L, rows, T;          // keys per head, proxy rows per row block (G*P, or 256 when G*P > 256), key tiles per head
  int rows_total, nrb;     // G*P and the number of 256-row blocks (1 unless G*P > 256)
  int Hkv;                 // kv heads per batch element (K tensor-map coordinates)
  int heads, n_slots;      // n_slots: epilogue warps that share a proxy row in sweep S = partials per (row, piece): 2 if rows > 128, else 4
  int causal, P;           // NACL_FLAG_CAUSAL: proxy row r (i = r % P, prompt position L-P+i) sees keys j <= L-P+i
  long long N;             // heads * T
  float scale_log2;        // log2(e) / sqrt(d)
  float2* part;            // [MAX_GRID + heads, n_slots, rows]  (m, z) per piece, log2 domain
  const float* lse_in;     // optional [heads*rows], natural log: given row statistics (no sweep S)
  float* lse_out;          // optional [heads*rows], natural log
  float* imp;              // [heads, L]
  float* imp_out;          // optional
  const int* table;        // paged K (or nullptr): page of position j of batch element hb = table[hb * tstride + j / ps]
  int ps, tstride;
  int* sync;               // fused launch: [2 * heads] zero at launch: per head the number of (CTA, row block) pieces whose
                           // partials are published, and the number of consumers that have seen them all (the last one
                           // zeroes both again)
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
// 4-D tile load with an L2 eviction-priority hint (createpolicy)
__device__ __forceinline__ void tma_load_4d_hint(uint32_t dst, const CUtensorMap* tm, int c0, int c1, int c2, int c3, uint32_t bar,
                                                 uint64_t policy) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3, %4, %5}], [%6], %7;"
      ::"r"(dst), "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(bar), "l"(policy)
      : "memory");
}
__device__ __forceinline__ uint64_t l2_policy_evict_first() {
  uint64_t p;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
  return p;
}

// one lane of the (converged) warp; the role loops run warp-wide so that addresses and descriptors stay in
// uniform registers, and only the TMA / MMA / commit instructions themselves are issued by the elected lane
__device__ __forceinline__ bool elect_one() {
  uint32_t pred;
  asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(pred));
  return pred != 0;
}

__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
// D[tmem] (+)= A[smem] * B[smem]^T, bf16 inputs, fp32 accumulate; issued by ONE thread
__device__ __forceinline__ void tc_mma(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
#ifdef NACL_DIAG_NO_MMA
  return;
#endif
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

__device__ __forceinline__ void tmem_ld8(uint32_t taddr, uint32_t (&v)[32]) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
               : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7])
               : "r"(taddr)
               : "memory");
}
__device__ __forceinline__ void tmem_ld4(uint32_t taddr, uint32_t (&v)[32]) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];"
               : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3])
               : "r"(taddr)
               : "memory");
}

__device__ __forceinline__ float fast_exp2(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}


typedef unsigned long long u64;
__device__ __forceinline__ u64 pack2(float a, float b) { u64 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b)); return r; }
__device__ __forceinline__ u64 pack2u(uint32_t a, uint32_t b) { u64 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "r"(a), "r"(b)); return r; }
__device__ __forceinline__ void unpack2(u64 r, float& a, float& b) { asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(r)); }
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c) { u64 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
__device__ __forceinline__ u64 add2(u64 a, u64 b) { u64 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ u64 sub2(u64 a, u64 b) { u64 r; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ u64 fma2_rm(u64 a, u64 b, u64 c) { u64 r; asm("fma.rm.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
__device__ __forceinline__ float fma_sat(float a, float b, float c) { float r; asm("fma.rn.sat.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c)); return r; }
__device__ __forceinline__ float max3(float a, float b, float c) { float r; asm("max.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c)); return r; }

// (2^x0, 2^x1) on the MUFU unit
__device__ __forceinline__ u64 exp2_mufu2(u64 x) {
  float a, b;
  unpack2(x, a, b);
  return pack2(fast_exp2(a), fast_exp2(b));
}
// acc += (2^x0, 2^x1) on the FMA pipe, for x = s*sc - ref given as the raw logits s and the two constants
//   scy = sc / 227,  cy = (127 - ref) / 227:
// y = sat(s*scy + cy) in [0, 1] IS the clamp of x to [-127, 100] (one saturating FMA, no min/max); u = 227*y = x + 127 in
// [0, 227]; n = floor(u) by a round-down FMA onto 1.5*2^23, f = u - n in [0, 1]; 2^f by the degree-3 minimax polynomial
// (relative error <= 7.5e-5); 2^(n-127) is the float whose exponent FIELD is n -- one shift -- multiplied in by the FMA that
// accumulates.  n = 0 (x < -126, or cy = -inf for a masked row) gives the scale +0.0: an exact zero, as MUFU.EX2.FTZ gives
// there.  x > 100 saturates at 2^100, which sweep S turns into a new reference (s_lazy32).  y resolves x to
// 227 * 2^-24 = 1.4e-5, i.e. 1e-5 relative in 2^x.  8 FMA-pipe instructions and 2 shifts per pair.
constexpr float kPolyLo = 127.f, kPolySpan = 227.f;
__device__ __forceinline__ u64 acc_exp2_poly_sat(u64 acc, uint32_t s0, uint32_t s1, float scy, float cy0, float cy1) {
  const u64 y = pack2(fma_sat(__uint_as_float(s0), scy, cy0), fma_sat(__uint_as_float(s1), scy, cy1));
  const u64 span = pack2(kPolySpan, kPolySpan), magic = pack2(12582912.f, 12582912.f);
  const u64 t = fma2_rm(y, span, magic);
  const u64 f = fma2(y, span, sub2(magic, t));  // 227*y - n
  u64 p = fma2(pack2(0.0780245f, 0.0780245f), f, pack2(0.22606719f, 0.22606719f));
  p = fma2(p, f, pack2(0.6958335f, 0.6958335f));
  p = fma2(p, f, pack2(0.9999252f, 0.9999252f));
  float t0, t1;
  unpack2(t, t0, t1);
  const u64 pw = pack2u(__float_as_uint(t0) << 23, __float_as_uint(t1) << 23);  // the magic constant's bits shift out: n << 23
  return fma2(p, pw, acc);
}
template <uint32_t MASK>
__device__ __forceinline__ constexpr bool pair_on_fma_pipe(int e) { return (MASK >> (e & 7)) & 1u; }

// lse (log2 domain) of one proxy row from its partials pp[c * stride], c < np, merged in ascending order with
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

// ------------------------------------------------------------------ the static schedule
// CTA c owns the flat tiles [N*c/G, N*(c+1)/G); sweep S walks them upwards, sweep C downwards.
// G*P > 256 (a multiple of 256): the proxy rows of a kv head are taken in blocks of 256; every segment is walked once per
// row block (rb = 0, 1, ...), its K tiles coming from L2 after the first time.
struct Seg { int head, tile, n, rb; };  // n tiles of `head`: tile, tile+step, ... (step = +1 in sweep S, -1 in sweep C); row block rb
struct Walk {
  long long t;
  int remaining, step, T, nrb, rb;
  Seg cur;
  __device__ Walk(const TcParams& p, int phase) {
    const long long G = gridDim.x, c = blockIdx.x;
    const long long t0 = p.N * c / G, t1 = p.N * (c + 1) / G;
    remaining = (int)(t1 - t0);
    step = phase ? -1 : 1;
    t = phase ? t1 - 1 : t0;
    T = p.T;
    nrb = p.nrb;
    rb = nrb;  // "current segment exhausted"
  }
  __device__ bool next(Seg& s) {
    if (rb < nrb) {  // the same tiles again, next row block
      cur.rb = rb++;
      s = cur;
      return true;
    }
    if (remaining <= 0) return false;
    cur.head = (int)(t / T);
    cur.tile = (int)(t - (long long)cur.head * T);
    const int room = step > 0 ? T - cur.tile : cur.tile + 1;
    cur.n = remaining < room ? remaining : room;
    cur.rb = 0;
    rb = 1;
    t += (long long)step * cur.n;
    remaining -= cur.n;
    s = cur;
    return true;
  }
};
// CTAs whose ranges contain the first / last tile of a head
__device__ __forceinline__ int cta_of_tile(long long t, long long N, long long G) { return (int)(((t + 1) * G + N - 1) / N - 1); }

// ------------------------------------------------------------------ shared-memory carve-up
// PH = the sweep the instantiation serves.  Sweep C carries two more operand boxes for the NINTH k-step of its MMAs (see
// "augmented contraction" at the kernel): QA = per proxy row the constant -lse/scale as three bf16 terms, KA = ones.
template <int QROWS, int NQ, int STAGES, int PH>
struct Smem {
  static constexpr int Q_BYTES = QROWS * HD * 2;
  static constexpr int QA_BYTES = QROWS * 128;  // one 128-byte (swizzled) row per proxy row; the first 32 bytes are used
  static constexpr int OFF_Q = 0;
  static constexpr int OFF_K = OFF_Q + NQ * Q_BYTES;
  static constexpr int OFF_QA = OFF_K + STAGES * KSTAGE_BYTES;
  static constexpr int OFF_KA = OFF_QA + (PH ? NQ * QA_BYTES : 0);
  static constexpr int OFF_CS = OFF_KA + (PH ? BOX_BYTES : 0);     // float[N_CS][4][128]: quarter column sums of a C tile
  static constexpr int OFF_BARS = OFF_CS + (PH ? N_CS * 4 * TILE * 4 : 0);
  static constexpr int N_BARS = 2 * STAGES + 4 * NQ + 4 * N_BUFS + 2 * N_CS + 2;  // (+2: partials of a segment stored / counted)
  static constexpr int OFF_TMEM = OFF_BARS + N_BARS * 8;
  static constexpr int TOTAL = OFF_TMEM + 8;
};

// ------------------------------------------------------------------ epilogue helpers
// max of 32 raw logits (3-input max, two chains)
__device__ __forceinline__ float s_max32(const uint32_t (&v)[32]) {
  float g0 = __uint_as_float(v[0]), g1 = __uint_as_float(v[1]);
#pragma unroll
  for (int e = 2; e < 30; e += 4) {
    g0 = max3(g0, __uint_as_float(v[e]), __uint_as_float(v[e + 2]));
    g1 = max3(g1, __uint_as_float(v[e + 1]), __uint_as_float(v[e + 3]));
  }
  return max3(g0, g1, fmaxf(__uint_as_float(v[30]), __uint_as_float(v[31])));
}
// (a0, a1) += 2^(v*sc - m_ref) over 32 columns, packed; some pairs on the FMA pipe (POLY_MASK)
__device__ __forceinline__ void s_acc32(const uint32_t (&v)[32], float sc, float m_ref, u64& a0, u64& a1) {
  const u64 sc2 = pack2(sc, sc), nm2 = pack2(-m_ref, -m_ref);
  const float scy = sc * (1.f / kPolySpan), cy = (kPolyLo - m_ref) * (1.f / kPolySpan);
#pragma unroll
  for (int e = 0; e < 16; e += 2) {
    if (pair_on_fma_pipe<NACL_POLY_MASK_S>(e)) a0 = acc_exp2_poly_sat(a0, v[2 * e + 0], v[2 * e + 1], scy, cy, cy);
    else a0 = add2(a0, exp2_mufu2(fma2(pack2u(v[2 * e + 0], v[2 * e + 1]), sc2, nm2)));
    if (pair_on_fma_pipe<NACL_POLY_MASK_S>(e + 1)) a1 = acc_exp2_poly_sat(a1, v[2 * e + 2], v[2 * e + 3], scy, cy, cy);
    else a1 = add2(a1, exp2_mufu2(fma2(pack2u(v[2 * e + 2], v[2 * e + 3]), sc2, nm2)));
  }
}
// one 32-column segment of an S tile: online (max, sum-exp) update of the row this thread owns
__device__ __forceinline__ void s_update(const uint32_t (&v)[32], float sc, float& m, float& z) {
#ifdef NACL_EPI_TRIVIAL  // diagnostics: pipeline ceiling without the exponentials (results are wrong)
  float t0 = 0.f;
#pragma unroll
  for (int e = 0; e < 32; ++e) t0 += __uint_as_float(v[e]);
  z += t0 * sc; m = 0.f;
  return;
#endif
  const float m_new = fmaxf(m, s_max32(v) * sc);
  u64 a0 = 0ull, a1 = 0ull;
  s_acc32(v, sc, m_new, a0, a1);
  float s0, s1;
  unpack2(add2(a0, a1), s0, s1);
  z = fmaf(z, fast_exp2(m - m_new), s0 + s1);
  m = m_new;
}
// Lazy reference (sweep S, full tiles).  The running sum is a plain fp32 sum of 2^(s*sc - m) for a reference m that
// stays where it is: fp32 keeps full relative accuracy for any m within ~100 (log2) of the values, so no running max
// and no rescale are needed per chunk.  Only when the sum leaves [0, 2^99) -- a value far above m, or the first chunk
// of a segment (m = -inf gives inf/NaN) -- the chunk is redone exactly with a new reference (s_update).  The pair
// (m, z) is a valid softmax partial for ANY finite m: merge_row never assumes that m is the true maximum.
__device__ __forceinline__ void s_lazy32(const uint32_t (&v)[32], float sc, float& m, float& z) {
#ifdef NACL_EPI_TRIVIAL
  s_update(v, sc, m, z);
  return;
#endif
  u64 a0 = 0ull, a1 = 0ull;
  s_acc32(v, sc, m, a0, a1);
  float s0, s1;
  unpack2(add2(a0, a1), s0, s1);
  const float zn = z + (s0 + s1);
  if (zn < 0x1p99f) {  // false for inf and NaN as well (the FMA-pipe exp2 saturates just below 2^100)
    z = zn;
  } else {
    s_update(v, sc, m, z);
    if (!(z < 0x1p99f)) { m += 90.f; z *= 0x1p-90f; }  // many terms just below the limit: move the reference, not the value
  }
}

// S tile, this warp's share: NC (32 or 64) key columns of the 32 proxy rows (TMEM lanes) it owns
// The accumulator buffer is handed back to the MMA warp (arrive on `empty_bar`) as soon as this warp's values are in
// registers, BEFORE the arithmetic: the MMAs of the tile after next start ~1500 cycles earlier.
__device__ __forceinline__ void release_tmem(uint32_t empty_bar) {
  tc_fence_before();
  __syncwarp();
  if ((threadIdx.x & 31) == 0) mbar_arrive(empty_bar);
}
template <int NC>
__device__ __forceinline__ void s_cols(uint32_t taddr, float sc, uint32_t empty_bar, float& m, float& z) {
  uint32_t va[32], vb[32];
  tmem_ld32(taddr, va);
  if (NC == 64) tmem_ld32(taddr + 32, vb);
  tc_wait_ld(va);
  if (NC == 64) tc_wait_ld(vb);
  release_tmem(empty_bar);
  s_lazy32(va, sc, m, z);
  if (NC == 64) s_lazy32(vb, sc, m, z);
}

// last tile of a head: columns >= valid (relative to taddr) are keys past L and must not exist (-inf)
// (warp-uniform `valid`: keys past L) and columns >= valid_t (per thread: keys its proxy row may not see, CAUSAL)
__device__ __forceinline__ void s_cols_masked(uint32_t taddr, int nc, float sc, int valid, int valid_t, float& m, float& z) {
  uint32_t v[32];
#pragma unroll 1
  for (int c = 0; c < nc && c < valid; c += 32) {
    tmem_ld32(taddr + c, v);
    tc_wait_ld(v);
    if (c < valid_t) {  // (a row with no visible key in this block keeps its statistics: max3 of all -inf would poison them)
#pragma unroll
      for (int e = 0; e < 32; ++e)
        if (c + e >= valid_t) v[e] = 0xFF800000u;
      s_update(v, sc, m, z);
    }
  }
}

// N4 groups of 4 columns (proxy rows) of a C tile: acc += 2^(v*sc), v = the accumulator, which already holds
// s - lse/scale (augmented contraction): no per-row constant, no shared-memory traffic in the epilogue
template <int N4>
__device__ __forceinline__ void c_update(const uint32_t (&v)[32], float sc, u64& a0, u64& a1) {
  const u64 sc2 = pack2(sc, sc), zero2 = 0ull;
  const float scy = sc * (1.f / kPolySpan), cy = kPolyLo * (1.f / kPolySpan);
#ifdef NACL_EPI_TRIVIAL
#pragma unroll
  for (int e = 0; e < N4; ++e) {
    a0 = add2(a0, pack2u(v[4 * e + 0], v[4 * e + 1]));
    a1 = add2(a1, pack2u(v[4 * e + 2], v[4 * e + 3]));
  }
  return;
#endif
#pragma unroll
  for (int e = 0; e < N4; ++e) {
    if (pair_on_fma_pipe<NACL_POLY_MASK_C>(2 * e)) a0 = acc_exp2_poly_sat(a0, v[4 * e + 0], v[4 * e + 1], scy, cy, cy);
    else a0 = add2(a0, exp2_mufu2(fma2(pack2u(v[4 * e + 0], v[4 * e + 1]), sc2, zero2)));
    if (pair_on_fma_pipe<NACL_POLY_MASK_C>(2 * e + 1)) a1 = acc_exp2_poly_sat(a1, v[4 * e + 2], v[4 * e + 3], scy, cy, cy);
    else a1 = add2(a1, exp2_mufu2(fma2(pack2u(v[4 * e + 2], v[4 * e + 3]), sc2, zero2)));
  }
}

// C tile, this warp's share: the key this thread owns, summed over nc proxy rows (TMEM columns from taddr on;
// nc a multiple of 4, <= 64) of exp2(v*sc)
__device__ __forceinline__ float c_cols(uint32_t taddr, int nc, float sc) {
  u64 a0 = 0ull, a1 = 0ull;
  uint32_t va[32], vb[32];
  if (nc == 64) {
    tmem_ld32(taddr, va);
    tmem_ld32(taddr + 32, vb);
    tc_wait_ld(va);
    c_update<8>(va, sc, a0, a1);
    tc_wait_ld(vb);
    c_update<8>(vb, sc, a0, a1);
  } else {
    int c = 0;
    if (nc & 32) { tmem_ld32(taddr, va); tc_wait_ld(va); c_update<8>(va, sc, a0, a1); c = 32; }
    if (nc & 16) { tmem_ld16(taddr + c, va); tc_wait_ld(va); c_update<4>(va, sc, a0, a1); c += 16; }
    if (nc & 8) { tmem_ld8(taddr + c, va); tc_wait_ld(va); c_update<2>(va, sc, a0, a1); c += 8; }
    if (nc & 4) { tmem_ld4(taddr + c, va); tc_wait_ld(va); c_update<1>(va, sc, a0, a1); }
  }
  float s0, s1;
  unpack2(add2(a0, a1), s0, s1);
  return s0 + s1;
}

// C tile under NACL_FLAG_CAUSAL (only the tiles that hold the last P keys): proxy rows r with r % P < imin do not see
// this thread's key and contribute nothing
__device__ __noinline__ float c_cols_causal(uint32_t taddr, int nc, float sc, int row0, int P, int imin) {
  float acc = 0.f;
  uint32_t v[32];
#pragma unroll 1
  for (int c = 0; c < nc; c += 4) {
    tmem_ld4(taddr + c, v);
    tc_wait_ld(v);
#pragma unroll
    for (int e = 0; e < 4; ++e)
      if ((row0 + c + e) % P >= imin) acc += fast_exp2(__uint_as_float(v[e]) * sc);
  }
  return acc;
}

// ------------------------------------------------------------------ inter-CTA hand-over of the partials (fused launch)
// Producer side (sweep S): see the publisher role in the kernel.
// Called by all epilogue threads before they read the partials of a head: one thread polls until all `need` pieces are
// published; the consumer that completes the head's `need` consumers zeroes both counters for the next launch.
__device__ __forceinline__ void await_pieces(int* cnt, int* done, int need) {
  if (threadIdx.x == 0) {
    uint32_t spins = 0;
    int v;
    do {
      asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(cnt) : "memory");
      if (++spins > SPIN_LIMIT) __trap();
    } while (v < need);
    if (atomicAdd(done, 1) == need - 1) {
      atomicExch(cnt, 0);
      atomicExch(done, 0);
    }
  }
  asm volatile("bar.sync 2, %0;" ::"n"(EPI_THREADS) : "memory");
}

// ------------------------------------------------------------------ the kernel
// One sweep (PH = 0: S, PH = 1: C) of the CTA's tile range.  Called once per sweep by the kernel below; TMEM is already
// allocated (tmem_base), the shared-memory carve-up and every mbarrier are (re)initialised here, and on return every
// asynchronous arrival on them has landed, so that the next sweep may carve the same bytes differently.
// FUSED: both sweeps run in one launch.  Sweep C of a head then needs the partials of every CTA whose range touches
// the head: a per-head counter in global memory (p.sync), incremented by each CTA once its partials of a segment are
// published and polled by one thread per consumer segment.  Nothing waits in sweep S, so the waits cannot form a cycle;
// the launch is cooperative, so every CTA is resident.
template <int QROWS, int NQ, int STAGES, int PH, bool FUSED>
__device__ __forceinline__ void sweep(const CUtensorMap& tmK, const CUtensorMap& tmQ, const TcParams& p, uint8_t* smem,
                                      const uint32_t sbase, const uint32_t tmem_base) {
  using SM = Smem<QROWS, NQ, STAGES, PH>;

  const uint32_t bars = sbase + SM::OFF_BARS;
  constexpr int B_KE = STAGES, B_QF = 2 * STAGES, B_QE = B_QF + NQ, B_AF = B_QE + NQ, B_AE = B_AF + NQ, B_TF = B_AE + NQ,
                B_TE = B_TF + 2 * N_BUFS, B_CF = B_TE + 2 * N_BUFS, B_CE = B_CF + N_CS;
  constexpr int B_PUB = B_CE + N_CS;
  static_assert(B_PUB + 2 == SM::N_BARS, "barrier count");
  // fused launch, sweep S: all epilogue warps have stored their partials of a segment / the publisher has taken note of it
  const uint32_t pub_bar = bars + 8u * B_PUB, pub_done = bars + 8u * (B_PUB + 1);
  auto qa_full = [&](int s) { return bars + 8u * (B_AF + s); };   // sweep C: the segment's -lse/scale rows are in shared memory
  auto qa_empty = [&](int s) { return bars + 8u * (B_AE + s); };  // ... and every MMA that read them has completed
  auto k_full = [&](int s) { return bars + 8u * s; };
  auto k_empty = [&](int s) { return bars + 8u * (B_KE + s); };
  auto q_full = [&](int s) { return bars + 8u * (B_QF + s); };
  auto q_empty = [&](int s) { return bars + 8u * (B_QE + s); };
  // accumulator barriers per (buffer, 128-row half): sweep S fills and drains the two halves of a tile independently,
  // sweep C (one N = G*P MMA group per tile) uses half 0 only
  auto tm_full = [&](int b, int h) { return bars + 8u * (B_TF + 2 * b + h); };
  auto tm_empty = [&](int b, int h) { return bars + 8u * (B_TE + 2 * b + h); };
  auto cs_full = [&](int b) { return bars + 8u * (B_CF + b); };
  auto cs_empty = [&](int b) { return bars + 8u * (B_CE + b); };
  float* cs_s = reinterpret_cast<float*>(smem + SM::OFF_CS);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int n_half = p.rows > 128 ? 2 : 1;  // 128-row MMA groups of an S tile
  // Quad accumulators (G*P > 128 in sweep S, G*P == 256 in sweep C).  The warp scheduler of an SM sub-partition prefers
  // one of its four epilogue warps, so they drift up to a tile apart; with whole-tile accumulators shared by all 16 warps
  // the slowest warp decides when a buffer goes back to the MMA issuer and the fast ones wait for the next tile.  Here a
  // tile's accumulator is produced and consumed as two independent 128-column halves (proxy rows 0..127 / 128..255 in
  // both sweeps: the 128-row MMA groups of sweep S, two N = 128 MMAs in sweep C), four half-buffers in all
  // (tile parity x half), each with its own full/empty barriers and its own FOUR consumers: the epilogue warps with
  // cq = 2 * (tile parity) + half, one per sub-partition and all of the same scheduling rank.  A warp processes 128
  // elements per thread of every other tile; while it waits for its half-buffer to be refilled (~900 cycles) the three
  // other ranks keep the sub-partition busy.
  const bool quad = PH == 0 ? p.rows > 128 : p.rows == 256;
  TR_DECL
  TL_DECL

  if (threadIdx.x == 0) {
    for (int s = 0; s < STAGES; ++s) { mbar_init(k_full(s), 1); mbar_init(k_empty(s), 1); }
    for (int s = 0; s < NQ; ++s) {
      mbar_init(q_full(s), 1); mbar_init(q_empty(s), 2);  // q_empty, qa_empty: one arrival per MMA issuer
      mbar_init(qa_full(s), 1); mbar_init(qa_empty(s), 2);
    }
    for (int b = 0; b < N_BUFS; ++b)
      for (int h = 0; h < 2; ++h) {
        mbar_init(tm_full(b, h), 1);
        mbar_init(tm_empty(b, h), quad ? 4 : N_EPI_WARPS);  // epilogue warps that drain it
      }
    for (int b = 0; b < N_CS; ++b) { mbar_init(cs_full(b), quad ? N_EPI_WARPS / 2 : N_EPI_WARPS); mbar_init(cs_empty(b), 1); }
    mbar_init(pub_bar, N_EPI_WARPS);
    mbar_init(pub_done, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if constexpr (PH != 0) {
    // KA: 128 key rows x 128 bytes in the operand layout (K-major, 128-byte swizzle: 16-byte chunk c of row r sits at chunk
    // c ^ (r & 7)); the k-step reads chunks 0 and 1 = 16 bf16 per row: {1, 1, 1, 0, ...}
    if (threadIdx.x < TILE) {
      const int r = threadIdx.x;
      uint4* row = reinterpret_cast<uint4*>(smem + SM::OFF_KA + r * 128);
      row[0 ^ (r & 7)] = make_uint4(0x3F803F80u, 0x00003F80u, 0u, 0u);
      row[1 ^ (r & 7)] = make_uint4(0u, 0u, 0u, 0u);
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // generic-proxy writes -> visible to the MMA's async proxy
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();

  if (warp == W_TMA) {
    // ================================================================ TMA producer
    const bool leader = elect_one();
    int stage = 0, qrun = 0, kuse = 0;
    uint32_t kphase = 0;
    // Every K tile is loaded with the L2 evict_first priority: K is a stream (268 MB per sweep at cfg 4 against 126 MB of L2),
    // and with the normal priority it pushes out what IS reused -- the importance row, the partials, Q, the rows the gather
    // is about to write.  Measured (us per call, same box): cfg 4 210.2 -> 207.2, cfg 3 108.5 -> 96.7, cfg 5 228 -> 217.2,
    // cfg 2 55.5 -> 53.9; keeping the tail of a CTA's sweep-S range with evict_last instead (16-110 MB) was worse than
    // hinting everything evict_first.
    const uint64_t pol_first = l2_policy_evict_first();
#ifdef NACL_DIAG_K_HINT  // diagnostics: bit 0 = hint in sweep S, bit 1 = in sweep C; without a hint: evict_normal
    uint64_t pol_normal;
    asm volatile("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(pol_normal));
    const uint64_t pol_k = ((NACL_DIAG_K_HINT >> PH) & 1) ? pol_first : pol_normal;
#else
    const uint64_t pol_k = pol_first;
#endif
    Walk walk(p, PH);
    Seg sg;
    while (walk.next(sg)) {
      const int qb = qrun % NQ;
      TRW(1, mbar_wait(q_empty(qb), ((qrun / NQ) & 1) ^ 1));
      const uint32_t qdst = sbase + SM::OFF_Q + qb * SM::Q_BYTES;
      if (leader) {
        mbar_expect_tx(q_full(qb), SM::Q_BYTES);
        tma_load_2d(qdst, &tmQ, 0, sg.head * p.rows_total + sg.rb * 256, q_full(qb));
        tma_load_2d(qdst + QROWS * 128, &tmQ, 64, sg.head * p.rows_total + sg.rb * 256, q_full(qb));
      }
      ++qrun;
      const int hb = sg.head / p.Hkv, hk = sg.head - hb * p.Hkv;  // K is addressed as [batch, kv head, key, d] with its own strides
      for (int i = 0; i < sg.n; ++i) {
        TRW(0, mbar_wait(k_empty(stage), kphase ^ 1));
        const uint32_t kdst = sbase + SM::OFF_K + stage * KSTAGE_BYTES;
#ifdef NACL_DIAG_SAME_TILE  // diagnostics: every K tile comes from L2 (results are wrong)
        const int j0 = ((sg.tile + walk.step * i) & 7) * TILE;
#elif defined(NACL_DIAG_RR_TILES)  // diagnostics: the CTAs stream one sliding window (tile = CTA + grid * step; results are wrong)
        const long long rr_ = ((long long)blockIdx.x + (long long)gridDim.x * kuse) % p.N;
        const int j0 = (int)(rr_ % p.T) * TILE;
        const int hh_ = (int)(rr_ / p.T);
        const int hb = hh_ / p.Hkv, hk = hh_ - hb * p.Hkv;
#else
        const int j0 = (sg.tile + walk.step * i) * TILE;
#endif
        if (p.table) {
          // paged K: the tile's 128 / ps pages are looked up by one lane each and loaded page by page into their rows of the
          // stage (ps rows x 128 B per box and page: a multiple of the 1024-byte swizzle atom).  Pages past the last key are
          // not loaded: their rows hold stale bytes, the keys past L are masked in both sweeps.
          const int nsub = TILE / p.ps;
          const int jb = j0 + lane * p.ps;
          int pg = 0;
          if (lane < nsub && jb < p.L) pg = __ldg(&p.table[(size_t)hb * p.tstride + jb / p.ps]);
          const int nload = min(nsub, (p.L - j0 + p.ps - 1) / p.ps);
          if (leader) mbar_expect_tx(k_full(stage), (uint32_t)(nload * p.ps * 256));
          for (int sb = 0; sb < nload; ++sb) {
            const int page = __shfl_sync(0xffffffffu, pg, sb);
            if (leader) {
              tma_load_4d_hint(kdst + sb * p.ps * 128, &tmK, 0, 0, hk, page, k_full(stage), pol_first);
              tma_load_4d_hint(kdst + BOX_BYTES + sb * p.ps * 128, &tmK, 64, 0, hk, page, k_full(stage), pol_first);
            }
          }
        } else if (leader) {
          mbar_expect_tx(k_full(stage), KSTAGE_BYTES);
          tma_load_4d_hint(kdst, &tmK, 0, j0, hk, hb, k_full(stage), pol_k);
          tma_load_4d_hint(kdst + BOX_BYTES, &tmK, 64, j0, hk, hb, k_full(stage), pol_k);
        }
        if (++stage == STAGES) { stage = 0; kphase ^= 1; }
        ++kuse;
      }
    }
    // drain: the tcgen05.commit arrivals on k_empty / q_empty / qa_empty of the last uses are asynchronous and nobody has
    // waited for them yet; they must have landed before these bytes are re-initialised or carved up differently
    for (int u = kuse > STAGES ? kuse - STAGES : 0; u < kuse; ++u) mbar_wait(k_empty(u % STAGES), (u / STAGES) & 1);
    for (int u = qrun > NQ ? qrun - NQ : 0; u < qrun; ++u) {
      mbar_wait(q_empty(u % NQ), (u / NQ) & 1);
      if constexpr (PH != 0) mbar_wait(qa_empty(u % NQ), (u / NQ) & 1);
    }
    __syncwarp();
  } else if (warp == W_MMA || warp == W_MMA2) {
    // ================================================================ tcgen05.mma issuers
    // Two issuer warps alternate tiles: issuer `mine` owns the tiles of that parity and the accumulator buffer of the
    // same number.  A tcgen05.mma issue blocks until the pipe has room, so one issuer spends the whole MMA time of a
    // tile inside the issue sequence; the other meanwhile sits through the barrier waits of the next tile (~200 cycles
    // each even when complete) and its MMAs queue up directly behind -- the tensor pipe no longer idles between tiles.
    const uint32_t mine = (uint32_t)(warp - W_MMA);
    const bool leader = elect_one();  // ONE lane issues every MMA and every commit (a commit covers its own thread's MMAs)
    int stage = 0, qrun = 0;
    uint32_t kphase = 0, tcount = 0;
    const uint32_t idesc = PH == 0 ? umma_idesc(128, TILE) : umma_idesc(128, p.rows);
    Walk walk(p, PH);
    Seg sg;
    while (walk.next(sg)) {
      const int qb = qrun % NQ;
      TRW(2, mbar_wait(q_full(qb), (qrun / NQ) & 1));
      if constexpr (PH != 0) {
        TRW(2, mbar_wait(qa_full(qb), (qrun / NQ) & 1));
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      }
      const uint32_t qsrc = sbase + SM::OFF_Q + qb * SM::Q_BYTES;
      const uint32_t qasrc = sbase + SM::OFF_QA + qb * SM::QA_BYTES, kasrc = sbase + SM::OFF_KA;
      ++qrun;
      if (sg.n == 1 && (tcount & 1) != mine) {
        // no tile of this segment is this issuer's: it still owes its arrival on q_empty (and qa_empty)
        if (leader) {
          mbar_arrive(q_empty(qb));
          if constexpr (PH != 0) mbar_arrive(qa_empty(qb));
        }
        __syncwarp();
      }
      for (int i = 0; i < sg.n; ++i) {
        const uint32_t buf = tcount & 1, par = (tcount >> 1) & 1;
        if (buf == mine) {
          TL(0)
          // An issuer sees only every other use of a stage when the ring length is odd, and a parity wait cannot tell
          // "this use has landed" from "the use before it has not even landed yet".  The consumer of the previous use (the
          // other issuer) commits k_empty only after that use's MMAs, so once k_empty has completed for it, k_full can
          // only be in the phase this tile needs.
          TRW(0, mbar_wait(k_empty(stage), kphase ^ 1));
          TRW(0, mbar_wait(k_full(stage), kphase));
          TL(1)
          const uint32_t ksrc = sbase + SM::OFF_K + stage * KSTAGE_BYTES;
          const uint32_t dcol = tmem_base + buf * BUF_COLS;
          if (quad) {
            // the two 128-column halves of the tile: each goes out as soon as ITS half-buffer is free
            const uint32_t idesc_q = umma_idesc(128, 128);
            for (uint32_t h = 0; h < 2; ++h) {
              TRW(1, mbar_wait(tm_empty(buf, h), par ^ 1));
              tc_fence_after();
              if (leader) {
#pragma unroll
                for (int k = 0; k < 8; ++k) {
                  const uint32_t ko = (k >> 2) * BOX_BYTES + (k & 3) * 32;
                  // proxy rows [128h, 128h+128) sit 128 rows x 128 B further down in each Q box
                  const uint32_t qo = (k >> 2) * (QROWS * 128) + (k & 3) * 32 + h * BOX_BYTES;
                  if constexpr (PH == 0) tc_mma(dcol + h * 128, umma_desc(qsrc + qo), umma_desc(ksrc + ko), idesc_q, k > 0);
                  else tc_mma(dcol + h * 128, umma_desc(ksrc + ko), umma_desc(qsrc + qo), idesc_q, k > 0);
                }
                // ninth k-step (sweep C): + ones x (-lse/scale) -- the row constant of the softmax goes in with the logits
                if constexpr (PH != 0) tc_mma(dcol + h * 128, umma_desc(kasrc), umma_desc(qasrc + h * BOX_BYTES), idesc_q, 1);
                tc_commit(tm_full(buf, h));
              }
              __syncwarp();
            }
            TL(2)
            if (leader) {
              tc_commit(k_empty(stage));
              if (i + 2 >= sg.n) {
                tc_commit(q_empty(qb));
                if constexpr (PH != 0) tc_commit(qa_empty(qb));
              }
            }
          } else {
          TRW(1, mbar_wait(tm_empty(buf, 0), par ^ 1));
          TL(2)
          tc_fence_after();
          if (leader) {
            if constexpr (PH == 0) {
              // the two 128-row halves accumulate into different TMEM columns: their k-steps are interleaved so that
              // consecutive MMAs never depend on each other (a dependent N=128 MMA chain runs at ~55 % of the pipe rate)
#pragma unroll
              for (int k = 0; k < 8; ++k) {
                const uint32_t ko = (k >> 2) * BOX_BYTES + (k & 3) * 32;
                const uint32_t qo = (k >> 2) * (QROWS * 128) + (k & 3) * 32;
                tc_mma(dcol, umma_desc(qsrc + qo), umma_desc(ksrc + ko), idesc, k > 0);
                if (n_half == 2) tc_mma(dcol + 128, umma_desc(qsrc + qo + BOX_BYTES), umma_desc(ksrc + ko), idesc, k > 0);
              }
            } else {
#pragma unroll
              for (int k = 0; k < 8; ++k) {
                const uint32_t ko = (k >> 2) * BOX_BYTES + (k & 3) * 32;
                const uint32_t qo = (k >> 2) * (QROWS * 128) + (k & 3) * 32;
                tc_mma(dcol, umma_desc(ksrc + ko), umma_desc(qsrc + qo), idesc, k > 0);
              }
              tc_mma(dcol, umma_desc(kasrc), umma_desc(qasrc), idesc, 1);  // ninth k-step: the row constants
            }
            tc_commit(tm_full(buf, 0));   // the accumulator buffer is complete
            tc_commit(k_empty(stage));    // the reads of the stage are done once these MMAs complete
            if (i + 2 >= sg.n) {          // this issuer's last tile of the segment: its reads of Q are done
              tc_commit(q_empty(qb));
              if constexpr (PH != 0) tc_commit(qa_empty(qb));
            }
          }
          }
          __syncwarp();
          TL(3)
          TL_NEXT()
        }
        ++tcount;
        if (++stage == STAGES) { stage = 0; kphase ^= 1; }
      }
    }
    __syncwarp();
  } else if (warp == W_CMB) {
    // ================================================================ sweep S of the fused launch: publisher of the partials
    // The epilogue warps only ARRIVE (mbarrier, release at CTA scope) once their partials of a segment are stored and go
    // on with the next segment; this otherwise idle warp waits for the 16 arrivals (acquire), makes the stores visible at
    // gpu scope and counts the piece.  (A __threadfence inside an epilogue warp stalled the accumulator hand-over for
    // 3-9 k cycles at every head boundary under a saturated memory system: profiles/r2b_final_kernels.md.)
    if constexpr (PH == 0 && FUSED) {
      uint32_t nseg = 0;
      Walk walk(p, PH);
      Seg sg;
      while (walk.next(sg)) {
        mbar_wait(pub_bar, nseg & 1);
        if (lane == 0) {
          mbar_arrive(pub_done);
          __threadfence();
          atomicAdd(p.sync + sg.head, 1);
        }
        __syncwarp();
        ++nseg;
      }
    }
    // ================================================================ column-sum combiner (sweep C only)
    if constexpr (PH != 0) {
      uint32_t ccount = 0;
      Walk walk(p, PH);
      Seg sg;
      while (walk.next(sg)) {
        for (int i = 0; i < sg.n; ++i, ++ccount) {
          const int cb = ccount % N_CS;
          TRW(0, mbar_wait(cs_full(cb), (ccount / N_CS) & 1));
          const float* c = cs_s + cb * 4 * TILE;
          float r[4];
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            const int key = lane + 32 * u;
            r[u] = quad ? c[key] + c[TILE + key] : (c[key] + c[TILE + key]) + (c[2 * TILE + key] + c[3 * TILE + key]);
          }
          __syncwarp();
          if (lane == 0) mbar_arrive(cs_empty(cb));
          const int j0 = (sg.tile - i) * TILE;
          const size_t o = (size_t)sg.head * p.L + j0;
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            const int key = lane + 32 * u;
            if (j0 + key < p.L) {
              // later row blocks add onto the sum of the earlier ones (same thread, same order every run)
              const float v = sg.rb == 0 ? r[u] : p.imp[o + key] + r[u];
              p.imp[o + key] = v;
              if (p.imp_out) p.imp_out[o + key] = v;
            }
          }
        }
      }
    }
  } else {
    // ================================================================ epilogue warps
    const int quarter = warp & 3, cq = warp >> 2;       // TMEM lane quarter, column quarter of the tile
    const uint32_t tbase = tmem_base + ((uint32_t)(quarter * 32) << 16);
    const float sc = p.scale_log2;
    const long long G = gridDim.x;
    // sweep S: this warp's proxy rows and key columns
    const int s_half = n_half == 2 ? (cq >> 1) : 0;
    const int s_slot = n_half == 2 ? (cq & 1) : cq;
    const int s_nc = n_half == 2 ? 64 : 32;
    const int s_col0 = s_slot * s_nc;
    const int s_row = s_half * 128 + quarter * 32 + lane;
    const bool live = s_half * 128 + quarter * 32 < p.rows;  // does this warp own a live proxy row?
    // sweep C: this warp's proxy rows (columns)
    const int c_nc = p.rows >> 2, c_col0 = cq * c_nc;
    // quad scheme: half and tile parity of this warp's half-buffer; the proxy row it owns in sweep S
    const int q_half = cq & 1, q_par = cq >> 1;
    const int q_row = q_half * 128 + quarter * 32 + lane;
    // G*P > 256 off the 256 grid: the last row block is partial.  Its MMA still runs 256 rows wide (the rows past the
    // head's G*P come from the next head or are zero-filled by the TMA: finite, and ignored below)
    auto rows_in_block = [&](int rb) { return min(p.rows, p.rows_total - rb * 256); };
    uint32_t ecount = 0;  // tiles seen so far, same sequence as the MMA warp's tcount
    int nseg = 0;
    Walk walk(p, PH);
    Seg sg;
    while (walk.next(sg)) {
      if constexpr (PH == 0) {
        // ---------------- S segment: running (reference, sum-exp) of row s_row over this warp's key columns
        float m0 = -INFINITY, z0 = 0.f;
        if (quad) {
          // this warp: proxy rows of half q_half (one per thread), all 128 key columns of the tiles of parity q_par
          for (int i = 0; i < sg.n; ++i) {
            const uint32_t g = ecount + i;
            if ((int)(g & 1) != q_par) continue;
            TL(0)
            TRW(0, mbar_wait(tm_full(q_par, q_half), (g >> 1) & 1));
            TL(1)
            tc_fence_after();
            const int valid = p.L - (sg.tile + i) * TILE;
            const bool ctile = p.causal && (sg.tile + i) * TILE + TILE - 1 > p.L - p.P;
            const uint32_t ta = tbase + q_par * BUF_COLS + q_half * 128;
            const uint32_t ebar = tm_empty(q_par, q_half);
            // warp-uniform (the TMEM loads are warp-wide): does this warp own a live proxy row of this row block?  Threads
            // past the last row compute on garbage and never store their statistics.
            const bool row_ok = q_half * 128 + quarter * 32 < rows_in_block(sg.rb);
            TRW(1, if (row_ok && !ctile && valid >= TILE) {
              uint32_t va[32], vb[32];
              tmem_ld32(ta, va);
              tmem_ld32(ta + 32, vb);
              tc_wait_ld(va);
              tc_wait_ld(vb);
              s_lazy32(va, sc, m0, z0);
              s_lazy32(vb, sc, m0, z0);
              tmem_ld32(ta + 64, va);
              tmem_ld32(ta + 96, vb);
              tc_wait_ld(va);
              tc_wait_ld(vb);
              release_tmem(ebar);  // the half-buffer goes back before the arithmetic on its last columns
              s_lazy32(va, sc, m0, z0);
              s_lazy32(vb, sc, m0, z0);
            } else {
              if (row_ok) {
                if (ctile) s_cols_masked(ta, TILE, sc, valid, min(valid, valid - p.P + 1 + (sg.rb * 256 + q_row) % p.P), m0, z0);
                else s_cols_masked(ta, TILE, sc, valid, valid, m0, z0);
              }
              release_tmem(ebar);
            })
            TL(2)
            TL_NEXT()
          }
          if (q_row < rows_in_block(sg.rb))
            __stcg(&p.part[(((size_t)blockIdx.x + sg.head) * p.n_slots + q_par) * p.rows_total + sg.rb * 256 + q_row], make_float2(m0, z0));
          if constexpr (FUSED) {
          // (a warp arrives for a segment only after the publisher has consumed the arrivals of the segment before it: the
          // publisher can never be two phases behind, however short the segments are)
          __syncwarp();
          if (lane == 0) {
            if (nseg > 0) mbar_wait(pub_done, (uint32_t)(nseg - 1) & 1u);
            mbar_arrive(pub_bar);
          }
        }
          ecount += sg.n;
          ++nseg;
          continue;
        }
        for (int i = 0; i < sg.n; ++i) {
          const uint32_t g = ecount + i, buf = g & 1;
          TRW(0, mbar_wait(tm_full(buf, 0), (g >> 1) & 1));
          tc_fence_after();
          const int valid = p.L - (sg.tile + i) * TILE - s_col0;
          // CAUSAL: this thread's row (i = s_row % P) sees the columns whose key j <= L-P+i
          const bool ctile = p.causal && (sg.tile + i) * TILE + TILE - 1 > p.L - p.P;
          const uint32_t ebar = tm_empty(buf, 0);
          TRW(1, if (live && !ctile && valid >= s_nc) {
            const uint32_t ta = tbase + buf * BUF_COLS + s_half * 128 + s_col0;
            if (n_half == 2) s_cols<64>(ta, sc, ebar, m0, z0); else s_cols<32>(ta, sc, ebar, m0, z0);  // releases the buffer itself
          } else {
            if (live) {
              const uint32_t ta = tbase + buf * BUF_COLS + s_half * 128 + s_col0;
              if (ctile) s_cols_masked(ta, s_nc, sc, valid, min(valid, valid - p.P + 1 + (sg.rb * 256 + s_row) % p.P), m0, z0);
              else s_cols_masked(ta, s_nc, sc, valid, valid, m0, z0);
            }
            release_tmem(ebar);
          })
        }
        // this warp's partial of the piece; (-inf, 0) when it saw no valid key
        if (s_row < p.rows)
          __stcg(&p.part[(((size_t)blockIdx.x + sg.head) * p.n_slots + s_slot) * p.rows_total + sg.rb * 256 + s_row], make_float2(m0, z0));
        if constexpr (FUSED) {
          // (a warp arrives for a segment only after the publisher has consumed the arrivals of the segment before it: the
          // publisher can never be two phases behind, however short the segments are)
          __syncwarp();
          if (lane == 0) {
            if (nseg > 0) mbar_wait(pub_done, (uint32_t)(nseg - 1) & 1u);
            mbar_arrive(pub_bar);
          }
        }
      } else {
        // ---------------- C segment: merge the head's partials (ascending piece order) into lse, hand -lse/scale to the MMA
        // issuers as the operand of the ninth k-step (augmented contraction: the accumulator then holds s - lse/scale and
        // the epilogue needs no per-row constant -- in this orientation a thread meets all G*P rows, and fetching their
        // constants from shared memory cost 10 us per sweep at cfg 4), then column sums
        const int qs = nseg % NQ;
        TRW(2, {
          mbar_wait(qa_empty(qs), ((nseg / NQ) & 1) ^ 1);  // the MMAs of the segment that used this slot before are done
          if constexpr (FUSED) {
            const int c_first = cta_of_tile((long long)sg.head * p.T, p.N, G);
            const int c_last = cta_of_tile((long long)(sg.head + 1) * p.T - 1, p.N, G);
            await_pieces(p.sync + sg.head, p.sync + p.heads + sg.head, (c_last - c_first + 1) * p.nrb);
          }
          const int r = threadIdx.x;
          if (r < p.rows) {
            float cf;
            if (r >= rows_in_block(sg.rb)) {
              cf = -INFINITY;  // a row past the head's G*P: 2^(-inf) = 0 on both exponential paths
            } else {
              float l2;
              if (p.lse_in) {
                l2 = p.lse_in[(size_t)sg.head * p.rows_total + sg.rb * 256 + r] * 1.4426950408889634f;  // given (natural log) -> log2 domain
              } else {
                const int c_first = cta_of_tile((long long)sg.head * p.T, p.N, G);
                const int c_last = cta_of_tile((long long)(sg.head + 1) * p.T - 1, p.N, G);
                l2 = merge_row(p.part + ((size_t)(c_first + sg.head) * p.n_slots) * p.rows_total + sg.rb * 256 + r,
                               (c_last - c_first + 1) * p.n_slots, (size_t)p.rows_total);
              }
              // the CTA that owns the head's first tile publishes lse
              if (p.lse_out && sg.tile - (sg.n - 1) == 0) p.lse_out[(size_t)sg.head * p.rows_total + sg.rb * 256 + r] = l2 * 0.69314718055994530942f;
              cf = -l2 / sc;  // in units of the raw dot product
            }
            // three bf16 terms carry cf to 2^-24 relative (the products with 1.0 are exact, the MMA sums them in fp32)
            const __nv_bfloat16 hi = __float2bfloat16_rn(cf);
            const bool fin = cf > -INFINITY;
            const float r1 = fin ? cf - __bfloat162float(hi) : 0.f;
            const __nv_bfloat16 mid = __float2bfloat16_rn(r1);
            const __nv_bfloat16 lo = __float2bfloat16_rn(r1 - __bfloat162float(mid));
            uint4* row = reinterpret_cast<uint4*>(smem + SM::OFF_QA + qs * SM::QA_BYTES + r * 128);
            row[0 ^ (r & 7)] = make_uint4((uint32_t)__bfloat16_as_ushort(hi) | ((uint32_t)__bfloat16_as_ushort(mid) << 16),
                                          (uint32_t)__bfloat16_as_ushort(lo), 0u, 0u);
            row[1 ^ (r & 7)] = make_uint4(0u, 0u, 0u, 0u);
          }
          // writers' generic-proxy stores -> async proxy (the MMA reads shared memory through it), then the epilogue
          // warps meet at a named barrier and ONE thread tells the issuers
          asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
          asm volatile("bar.sync 1, %0;" ::"n"(EPI_THREADS) : "memory");
          if (threadIdx.x == 0) mbar_arrive(qa_full(qs));
        })
        if (quad) {
          // this warp: the 32 keys of its lane quarter (one per thread) summed over the 128 proxy rows of half q_half, for
          // the tiles of parity q_par; the combiner adds the two halves of a key
          for (int i = 0; i < sg.n; ++i) {
            const uint32_t g = ecount + i;
            if ((int)(g & 1) != q_par) continue;
            const int cb = g % N_CS;
            TL(0)
            TRW(0, mbar_wait(tm_full(q_par, q_half), (g >> 1) & 1));
            TL(1)
            tc_fence_after();
            const uint32_t ta = tbase + q_par * BUF_COLS + q_half * 128;
            const uint32_t ebar = tm_empty(q_par, q_half);
            float r;
            if (p.causal && (sg.tile - i) * TILE + TILE - 1 > p.L - p.P) {
              const int jkey = (sg.tile - i) * TILE + quarter * 32 + lane;  // the key this thread owns
              r = c_cols_causal(ta, 128, sc, sg.rb * 256 + q_half * 128, p.P, jkey - (p.L - p.P));
              release_tmem(ebar);
            } else {
              TRW(1, {
                u64 a0 = 0ull, a1 = 0ull;
                uint32_t va[32], vb[32];
                tmem_ld32(ta, va);
                tmem_ld32(ta + 32, vb);
                tc_wait_ld(va);
                c_update<8>(va, sc, a0, a1);
                tc_wait_ld(vb);
                c_update<8>(vb, sc, a0, a1);
                tmem_ld32(ta + 64, va);
                tmem_ld32(ta + 96, vb);
                tc_wait_ld(va);
                tc_wait_ld(vb);
                release_tmem(ebar);
                c_update<8>(va, sc, a0, a1);
                c_update<8>(vb, sc, a0, a1);
                float s0, s1;
                unpack2(add2(a0, a1), s0, s1);
                r = s0 + s1;
              })
            }
            TL(2)
            TRW(4, mbar_wait(cs_empty(cb), ((g / N_CS) & 1) ^ 1));
            cs_s[(cb * 4 + q_half) * TILE + quarter * 32 + lane] = r;
            __syncwarp();
            if (lane == 0) mbar_arrive(cs_full(cb));
            TL(3)
            TL_NEXT()
          }
          ecount += sg.n;
          ++nseg;
          continue;
        }
        for (int i = 0; i < sg.n; ++i) {
          const uint32_t g = ecount + i, buf = g & 1;
          const int cb = g % N_CS;
          TRW(0, mbar_wait(tm_full(buf, 0), (g >> 1) & 1));
          tc_fence_after();
          float r;
          const int jkey = (sg.tile - i) * TILE + quarter * 32 + lane;  // the key this thread owns
          if (p.causal && (sg.tile - i) * TILE + TILE - 1 > p.L - p.P)
            r = c_cols_causal(tbase + buf * BUF_COLS + c_col0, c_nc, sc, sg.rb * 256 + c_col0, p.P, jkey - (p.L - p.P));
          else
            TRW(1, r = c_cols(tbase + buf * BUF_COLS + c_col0, c_nc, sc));
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(tm_empty(buf, 0));
          TRW(4, mbar_wait(cs_empty(cb), ((g / N_CS) & 1) ^ 1));
          cs_s[(cb * 4 + cq) * TILE + quarter * 32 + lane] = r;
          __syncwarp();
          if (lane == 0) mbar_arrive(cs_full(cb));
        }
      }
      ecount += sg.n;
      ++nseg;
    }
  }

  TR_FLUSH()
  tc_fence_before();
  __syncthreads();
}

// MODE 0: sweep S, 1: sweep C (two launches, or lse_in given), 2: S then C in one cooperative launch
template <int QROWS, int NQ, int STAGES_S, int STAGES_C, int MODE>
__global__ void __launch_bounds__(NTHREADS, 1)
nacl_score_tc_kernel(const __grid_constant__ CUtensorMap tmK, const __grid_constant__ CUtensorMap tmQ, const TcParams p) {
  extern __shared__ __align__(1024) uint8_t smem[];
  const uint32_t sbase = smem_u32(smem);
  if ((sbase & 1023u) != 0) __trap();  // the 128B-swizzled operand tiles need 1024-byte alignment
  GSTAMP(0)
  __shared__ uint32_t tmem_slot;
  const int warp = threadIdx.x >> 5;
  if (warp == W_MMA) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_slot)), "r"(TMEM_COLS) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *reinterpret_cast<volatile uint32_t*>(&tmem_slot);
  GSTAMP(1)
  if constexpr (MODE != 1) sweep<QROWS, NQ, STAGES_S, 0, MODE == 2>(tmK, tmQ, p, smem, sbase, tmem_base);
  GSTAMP(2)
  if constexpr (MODE != 0) sweep<QROWS, NQ, STAGES_C, 1, MODE == 2>(tmK, tmQ, p, smem, sbase, tmem_base);
  GSTAMP(3)
  if (warp == W_MMA) {
    tc_fence_after();
    __syncwarp();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(TMEM_COLS) : "memory");
  }
}

// Sweep S on its own (nacl_proxy_lse): lse of every proxy row from the partials that a MODE 0 launch of `grid` CTAs left,
// merged exactly as the column-sum sweep merges them (same routine, same ascending piece order: the same bits).
__global__ void __launch_bounds__(128) nacl_lse_merge_kernel(const float2* __restrict__ part, float* __restrict__ lse_out, int rows_total,
                                                             int T, long long N, int grid, int n_slots) {
  const int head = blockIdx.y;
  const int r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= rows_total) return;
  const int c_first = cta_of_tile((long long)head * T, N, grid);
  const int c_last = cta_of_tile((long long)(head + 1) * T - 1, N, grid);
  const float l2 = merge_row(part + ((size_t)(c_first + head) * n_slots) * rows_total + r, (c_last - c_first + 1) * n_slots, (size_t)rows_total);
  lse_out[(size_t)head * rows_total + r] = l2 * 0.69314718055994530942f;
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

template <class Kern>
cudaError_t launch_one(Kern kern, int grid, int smem_bytes, bool cooperative, const CUtensorMap& tmK, const CUtensorMap& tmQ,
                       const TcParams& p, cudaStream_t st) {
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes);
  if (e != cudaSuccess) return e;
  cudaLaunchConfig_t cfg = {};
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeCooperative;  // every CTA resident: the fused launch has inter-CTA waits
  attr[0].val.cooperative = 1;
  cfg.gridDim = dim3((unsigned)grid);
  cfg.blockDim = dim3(NTHREADS);
  cfg.dynamicSmemBytes = (size_t)smem_bytes;
  cfg.stream = st;
  cfg.attrs = attr;
  cfg.numAttrs = cooperative ? 1 : 0;
  return cudaLaunchKernelEx(&cfg, kern, tmK, tmQ, p);
}

template <int QROWS, int NQ, int STAGES_S, int STAGES_C>
cudaError_t launch_cfg(const CUtensorMap& tmK, const CUtensorMap& tmQ, TcParams p, bool two_launches, bool stats_only, cudaStream_t st) {
  using SMS = Smem<QROWS, NQ, STAGES_S, 0>;
  using SMC = Smem<QROWS, NQ, STAGES_C, 1>;
  constexpr int kStatic = 1024 + 16;  // the kernel's static shared memory (TMEM slot) and the alignment gap it may cause
  static_assert(SMS::TOTAL + kStatic <= 227 * 1024 && SMC::TOTAL + kStatic <= 227 * 1024, "shared memory budget");
  constexpr int kBoth = SMS::TOTAL > SMC::TOTAL ? SMS::TOTAL : SMC::TOTAL;
  long long grid = sm_count() < MAX_GRID ? sm_count() : MAX_GRID;
  if (p.N < grid) grid = p.N;
  cudaError_t e;
  if (stats_only) {  // the statistics sweep, then the merge of its partials into lse_out: no column sums
    {
      StageScope sc(ST_STATS, st);
      e = launch_one(nacl_score_tc_kernel<QROWS, NQ, STAGES_S, STAGES_C, 0>, (int)grid, SMS::TOTAL, false, tmK, tmQ, p, st);
      if (e != cudaSuccess) return e;
    }
    StageScope sc(ST_COMBINE, st);
    nacl_lse_merge_kernel<<<dim3((unsigned)((p.rows_total + 127) / 128), (unsigned)p.heads), 128, 0, st>>>(p.part, p.lse_out, p.rows_total, p.T, p.N,
                                                                                                        (int)grid, p.n_slots);
    return cudaGetLastError();
  }
  if (p.lse_in) {
    StageScope sc(ST_COLSUM, st);
    return launch_one(nacl_score_tc_kernel<QROWS, NQ, STAGES_S, STAGES_C, 1>, (int)grid, SMC::TOTAL, false, tmK, tmQ, p, st);
  }
  if (!two_launches) {
    StageScope sc(ST_FUSED, st);
    return launch_one(nacl_score_tc_kernel<QROWS, NQ, STAGES_S, STAGES_C, 2>, (int)grid, kBoth, true, tmK, tmQ, p, st);
  }
  {
    StageScope sc(ST_STATS, st);
    e = launch_one(nacl_score_tc_kernel<QROWS, NQ, STAGES_S, STAGES_C, 0>, (int)grid, SMS::TOTAL, false, tmK, tmQ, p, st);
    if (e != cudaSuccess) return e;
  }
  StageScope sc(ST_COLSUM, st);
  return launch_one(nacl_score_tc_kernel<QROWS, NQ, STAGES_S, STAGES_C, 1>, (int)grid, SMC::TOTAL, false, tmK, tmQ, p, st);
}

}  // namespace

bool score_tc_supported(const Shape& s) {
  return s.dtype == NACL_DTYPE_BF16 && s.d == HD && s.rows % 16 == 0 && s.rows >= 16 &&
         s.rows <= 8192;  // G*P > 256: blocks of 256 proxy rows, the last one masked where G*P is off that grid
}


size_t score_tc_part_elems(int heads, int rows) { return (size_t)(MAX_GRID + heads) * 4 * rows; }

cudaError_t launch_score_tc(const Shape& s, const void* K, const void* Q, const SplitPlan&, const Workspace& ws,
                            const float* lse_in, bool causal, bool two_launches, float* imp_out, float* lse_out, cudaStream_t st,
                            bool stats_only) {
  if (stats_only && (!lse_out || lse_in)) return cudaErrorInvalidValue;
  EncodeTiledFn enc = encode_tiled_fn();
  if (!enc) return cudaErrorNotSupported;  // no silent fallback: the caller reports NACL_ERR_CUDA
  const int heads = s.batch * s.Hkv;
  const int qrows = s.rows <= 128 ? 128 : 256;

  alignas(64) CUtensorMap tmK, tmQ;
  {
    // [batch, Hkv, L, d] with the caller's strides (contiguous, a cache with spare capacity, or token-major [B,L,H,d])
    // paged: [n_pages, Hkv, page_size, d] with the pool's strides, one box = the 64 columns of one page's rows
    const bool paged = s.table != nullptr;
    const cuuint64_t dims[4] = {(cuuint64_t)HD, (cuuint64_t)(paged ? s.ps : s.L), (cuuint64_t)s.Hkv, (cuuint64_t)(paged ? s.n_pages : s.batch)};
    const cuuint64_t strides[3] = {(cuuint64_t)s.kv_sr * 2, (cuuint64_t)s.kv_sh * 2, (cuuint64_t)(paged ? s.kv_sp : s.kv_sb) * 2};
    const cuuint32_t box[4] = {64, (cuuint32_t)(paged ? s.ps : TILE), 1, 1};
    const cuuint32_t es[4] = {1, 1, 1, 1};
#ifndef NACL_K_L2PROMO
#define NACL_K_L2PROMO CU_TENSOR_MAP_L2_PROMOTION_L2_256B
#endif
    if (enc(&tmK, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, const_cast<void*>(K), dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
            CU_TENSOR_MAP_SWIZZLE_128B, NACL_K_L2PROMO, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
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
  p.L = s.L; p.rows = s.rows <= 256 ? s.rows : 256; p.T = (s.L + TILE - 1) / TILE;
  p.rows_total = s.rows; p.nrb = (s.rows + 255) / 256;
  p.heads = heads; p.Hkv = s.Hkv;
  p.n_slots = s.rows <= 128 ? 4 : 2;
  p.causal = causal ? 1 : 0; p.P = s.P;
  p.N = (long long)heads * p.T;
  p.scale_log2 = 1.4426950408889634f / sqrtf((float)s.d);
  p.part = ws.part; p.lse_in = lse_in; p.lse_out = lse_out; p.imp = ws.imp; p.imp_out = imp_out;
  p.sync = ws.sync;
  p.table = s.table; p.ps = s.ps; p.tstride = s.tstride;
#ifndef NACL_STAGES_S
#define NACL_STAGES_S 5
#endif
  if (qrows == 128) return launch_cfg<128, 2, NACL_STAGES_S, 3>(tmK, tmQ, p, two_launches, stats_only, st);
  return launch_cfg<256, 1, NACL_STAGES_S, 3>(tmK, tmQ, p, two_launches, stats_only, st);
}

}  // namespace nacl

#ifdef NACL_TC_STAMPS
extern "C" __attribute__((visibility("default"))) int nacl_debug_stamps_read(long long* host) {
  return (int)cudaMemcpyFromSymbol(host, nacl::g_stamps, sizeof(nacl::g_stamps));
}
#endif
#ifdef NACL_TC_TRACE
// diagnostics build only: per-warp wait/compute cycle counters of the last launches
extern "C" __attribute__((visibility("default"))) int nacl_debug_trace_read(long long* host, size_t bytes) {
  return (int)cudaMemcpyFromSymbol(host, nacl::g_trace, bytes < sizeof(nacl::g_trace) ? bytes : sizeof(nacl::g_trace));
}
extern "C" __attribute__((visibility("default"))) int nacl_debug_timeline_read(long long* host) {
  return (int)cudaMemcpyFromSymbol(host, nacl::g_tl, sizeof(nacl::g_tl));
}
#endif
