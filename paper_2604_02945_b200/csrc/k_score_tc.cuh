// k_score_tc.cuh — the Blackwell fast path of the score pass (SURVEY.md §8(a) rows a0+a1+a2+a3 in ONE sweep over X),
// bf16 inputs with d % 64 == 0.
//
// Work unit = a TILE: up to 8 row BLOCKS (<= 128 rows each) of one segment that share the request's query rows, swept
// K-OUTERMOST: for every 64-column K-chunk the query chunk Q[L, kc] is staged once (TMA, small ring of its own) and every
// block's chunk X[rows_b, kc] streams through a ring of 16 KB slots (TMA, SWIZZLE_128B), each consumed by
//   * one elected thread issuing tcgen05.mma (kind::f16, bf16 x bf16 -> fp32, M = 128, N = pad16(L), 4 x K = 16) into the
//     block's own accumulator slot in TMEM: S = X·Q^T                                                   (Eq. 6)
//   * eight CUDA-core warps (two threads per row, half a 128-byte row each, conflict-free through the hardware swizzle)
//     accumulating sum x^2 and sum (x - x_prev)^2 with packed fp32x2 FMAs                         (Eq. 3, Eq. 5)
// and released by both.  Three kinds of tile:
//   mode 0  blocks = consecutive 128-row pieces of a single-frame segment (no temporal term);
//   mode 1  "frame walk": the blocks are the SAME patch rows in consecutive frames t0 .. t0+F-1.  The previous frame's
//           K-chunk of a row is simply the chunk the statistics thread read one block earlier, so it is carried in
//           REGISTERS: every byte of X enters shared memory once and no ring space is spent on previous-frame copies
//           (frame t0-1 rides along as a "halo" chunk that only the statistics warps read; an L2 hit);
//   mode 2  short frames (P < 64, e.g. audio with P = 1): blocks are overlapping 128-row windows, the previous-frame
//           row r - P sits in the same chunk.
// Four epilogue warps read the accumulator slots with tcgen05.ld (one token row per thread: the max over query tokens
// needs no shuffles), scale by 1/|q_j| and 1/|x_i| and write s, sqrt(D), rel: 12 B per token.  gamma = sqrt(D) / (|x_t| +
// |x_{t-1}|) is finished by the segment kernel, which has both norms from s.  The query norms (row a0) are computed by the
// epilogue warps while the first chunks stream in (grid-wide counter, cooperative launch).
// NEXT-1 / NEXT-2 riders: 64 hash rows or head-weight rows follow the query rows in the B tile (N = pad16(L) + 64).
//
// Persistent: one CTA per SM walks a host-built list of tiles cut to equal cost at single-row granularity.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <cstring>
#include <vector>

#include "../../include/msas.h"
#include "msas_internal.cuh"

namespace msas {

struct TcTile {            // 64 bytes
  int32_t row0;            // global row id of the first row block 0 loads
  int32_t n_rows;          // mode 1: rows of every block (<= 128); modes 0, 2: rows the tile loads in total (blocks of <= 128)
  int32_t n_blocks;        // 1..8 (<= TMEM accumulator slots)
  int32_t stride;          // rows between the first rows of consecutive blocks (mode 0: the block height <= 128, mode 1: P, mode 2: 128 - P)
  int32_t mode;            // see above
  int32_t prev;            // P for modes 1 and 2, else 0
  int32_t halo;            // mode 1: 1 = a halo chunk (frame t0 - 1) precedes the blocks of every K-chunk;
                           // mode 2: leading rows of block 0 that are loaded for their successors only (0 or P)
  int32_t q_row0;          // first query row of the request
  int32_t L;               // query tokens of the request
  int32_t part0;           // NEXT-2: slot of block 0's column sums (block b -> part0 + b); slots of a segment are contiguous
  int32_t seg;
  // K-split: CTAs may share a row block along K.  The tile's LAST block is swept over the K-chunks [k0, nk) only and its FIRST
  // block over [0, k1) only (a one-block tile: [k0, k1)); the blocks in between over all of K.  The part of a block that ends
  // at chunk nk OWNS it: it is the last thing its CTA does, and it adds the partial accumulators and row sums the other parts
  // dumped and writes the results.  A part with k1 < nk is the first block of its CTA's first tile: it is complete early in
  // that CTA's sweep and dumped into the exchange slot of the CTA right away, long before the owner asks for it.
  int32_t k0, k1;          // in 64-column chunks, multiples of the slices per chunk; 0 and nk where the tile is not split
  int32_t n_wait;          // owner (last block with k0 > 0, k1 = nk if it is the only one): number of foreign parts (exchange slots peer .. peer + n_wait - 1)
  int32_t peer;            // owner: first exchange slot to read (the CTA after this one); -1 otherwise
  int32_t pad_;
};
static_assert(sizeof(TcTile) == 64, "TcTile is 64 bytes");

constexpr int kTcThreads = 448;                      // 14 warps: 4 epilogue, 8 statistics, TMA producer, MMA issuer (144 registers per thread)
constexpr int kTcAluWarps = 8;
constexpr int kTcWarpTma = 12, kTcWarpMma = 13;
constexpr int kTcMaxCtas = 160;                     // CTAs of a launch (one per SM) = K-split exchange slots
constexpr int kTcMaxBlocks = 10;                    // blocks per tile = TMEM accumulator slots (512 columns / pad16(L), at most 10)
constexpr int kTcSliceBytes = 128 * 128;             // 128 rows x 64 bf16 columns: one K-slice of a block
constexpr int kTcMaxXSlots = 12;
constexpr int kTcCtrlBytes = 4096;
constexpr int kTcStatBytes = 2 * kTcMaxBlocks * 128 * 2 * 4;   // [buffer][block][row][n2, D]
constexpr int kTcSmemBytes = 227 * 1024;

struct TcMaps {
  CUtensorMap x[16];   // token rows as a 3-D tensor [d / 64 slices][N rows][64 columns]: box = kw slices x 8 * (i + 1) rows x 64 columns
  CUtensorMap q[3];    // query rows: box = 64 / 32 / 16 rows x 64 columns
  CUtensorMap r;       // riders: the 64 hash / head-weight rows R[64, d] (box = 64 rows x 64 columns)
};

struct TcSchedule {
  bool enabled = false;
  int n_ctas = 0, n_tiles = 0, n_parts = 0;
  int kw = 1;              // 64-column K-slices per chunk (2 where d % 128 == 0: half the barrier round trips per byte)
  int nx = 0;              // X ring slots (kw * 16 KB each)
  int qslot_bytes = 0;     // bytes of one query-chunk slot
  int nq = 2;              // query-chunk slots (2..4: short tiles need several K-steps in flight)
  int wslot = 0, ns = 0;        // TMEM: columns per accumulator slot (pad16 of the longest query block), number of slots
  int smem_bytes = 0;
  int xchg_cols = 0;       // floats per row of a K-split exchange slot: pad16(longest query block) (+ 64) + 2
  int help = 0;            // 1: the HELP instantiation of the kernel is launched
  const TcTile* d_tiles = nullptr;
  const int32_t* d_cta_off = nullptr;
};

struct TcParams {
  const TcTile* tiles;
  const int32_t* cta_off;
  float* qinv;                       // [nQ] 1 / |q_j|, written by this kernel's own prologue (a0) and read by its epilogues
  const void* Q;                     // query rows (bf16), for that prologue; NULL = qinv was computed by k_qprep before this launch
  long long nQ;
  unsigned long long* q_ready;       // [0] grid-wide arrival counter of the prologue, [1] CTAs that have left the kernel;
                                     // both zero between launches (the last CTA to leave re-arms them: graph-replay safe)
  unsigned long long* sig;           // NEXT-1 (literal LSH probe, Eq. 5): NULL = off; else the hash rows ride the MMA as 64 more B rows
  // NEXT-2 (learned heads, Eq. 3 / Eq. 6): NULL = off; else the 64 weight rows W ride the MMA like the hash rows (never both):
  // heads_m[row] = sigmoid(w_0 . x + heads_bias); heads_part[(part0 + b) * 64 + c] = per block of a tile, the number of rows
  // with heads_m < heads_tau (c = 0) and the column sums of w_c . x (c = 1..63)
  float* heads_part;
  float* heads_m;
  float heads_bias, heads_tau;
  float* s;
  float* dnorm;       // sqrt(sum (x - x_prev)^2) for rows that have a previous frame
  float* rel;
  int d;
  int n_kchunks;
  int kw, nx, nq, qslot_bytes, wslot, ns;
  float* xchg;            // K-split exchange: slot c = [xchg_cols][128] floats (accumulator columns, then sum x^2, sum (x - x_prev)^2)
  unsigned int* xflag;    // [n_ctas] 1 = slot c is filled; zero between launches (the owner re-arms it)
  int xchg_cols;
};

__device__ __forceinline__ int tc_block_rows(const TcTile& t, int b) {
  return t.mode == 1 ? t.n_rows : min(t.mode == 0 ? t.stride : 128, t.n_rows - b * t.stride);
}
// K-chunks a tile walks, and the blocks that take part in chunk kc: block 0 leaves at k1, the last block joins at k0
__device__ __forceinline__ int tc_k_lo(int n_blocks, int k0) { return n_blocks == 1 ? k0 : 0; }
__device__ __forceinline__ int tc_k_hi(int n_blocks, int k1, int nk) { return n_blocks == 1 ? k1 : nk; }
__device__ __forceinline__ int tc_b_first(int kc, int k1, int n_blocks) { return n_blocks > 1 && kc >= k1 ? 1 : 0; }
__device__ __forceinline__ int tc_b_end(int kc, int k0, int n_blocks) { return n_blocks > 1 && kc < k0 ? n_blocks - 1 : n_blocks; }

// ------------------------------------------------------------------------------------------------ PTX wrappers
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(bar), "r"(parity)
      : "memory");
}
__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap* map, uint32_t bar, int c0, int c1, int c2) {
  asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];" ::"r"(dst),
               "l"(map), "r"(bar), "r"(c0), "r"(c1), "r"(c2)
               : "memory");
}
// the same with an L2 eviction-priority hint (createpolicy): the bulk of X is read once and should not push the query rows,
// the halo frames and the exchange slots out of L2
__device__ __forceinline__ void tma_load_3d_hint(uint32_t dst, const CUtensorMap* map, uint32_t bar, int c0, int c1, int c2, uint64_t pol) {
  asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%3, %4, %5}], [%2], %6;" ::"r"(dst),
               "l"(map), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "l"(pol)
               : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void tc_mma_bf16(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "setp.ne.b32 p, %4, 0;\n"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n"
      "}\n" ::"r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ void tc_ld16(uint32_t taddr, uint32_t (&v)[16]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
      : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]), "=r"(v[9]),
        "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
      : "r"(taddr)
      : "memory");
}
__device__ __forceinline__ void tc_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// packed fp32 pairs (Blackwell FFMA2 / FADD2): two lanes of fp32 per 64-bit register
__device__ __forceinline__ uint64_t bf16x2_to_f32x2(uint32_t w) {   // exact: low half -> .x, high half -> .y
  uint64_t r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "r"(w << 16), "r"(w & 0xffff0000u));
  return r;
}
__device__ __forceinline__ uint64_t sub_f32x2(uint64_t a, uint64_t b) {
  uint64_t r;
  asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
__device__ __forceinline__ void fma_sq_f32x2(uint64_t& acc, uint64_t a) {   // acc += a * a (per lane)
  asm("fma.rn.f32x2 %0, %1, %1, %0;" : "+l"(acc) : "l"(a));
}
__device__ __forceinline__ float sum_f32x2(uint64_t a) {
  float lo, hi;
  asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(a));
  return lo + hi;
}

// shared-memory matrix descriptor: K-major, SWIZZLE_128B, 8-row groups 1024 B apart (sm_100 descriptor version 1)
__device__ __forceinline__ uint64_t umma_desc_sw128(uint32_t saddr) {
  const uint32_t lo = ((saddr & 0x3FFFFu) >> 4) | (1u << 16);             // start address | LBO (unused for swizzled K-major)
  const uint32_t hi = (1024u >> 4) | (1u << 14) | (2u << 29);             // SBO = 1024 B | version 1 | SWIZZLE_128B
  return ((uint64_t)hi << 32) | lo;
}
// instruction descriptor: D fp32, A/B bf16, both K-major, M = 128, N = n
__device__ __forceinline__ uint32_t umma_idesc_bf16(int n) {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(n >> 3) << 17) | ((128u >> 4) << 24);
}

// ------------------------------------------------------------------------------------------------ the kernel
struct TcCtrl {                      // lives at the (1024-aligned) start of dynamic shared memory
  uint64_t xfull[kTcMaxXSlots];      // TMA -> consumers           (1 arrival + transaction bytes)
  uint64_t xempty[kTcMaxXSlots];     // consumers -> TMA           (1 MMA commit + the statistics warps)
  uint64_t qfull[4], qempty[4];      // the query-chunk ring: TMA -> MMA, MMA commit -> TMA
  uint64_t tfull[kTcMaxBlocks];      // accumulator slot: MMA commit -> epilogue
  uint64_t tempty[kTcMaxBlocks];     // epilogue (4 warps) -> MMA
  uint64_t sfull[2], sempty[2];      // row statistics of a tile: statistics warps -> epilogue (4 warps) -> statistics warps
  uint64_t s0full;                   // row statistics of a dumped first block (at most one per CTA: single use)
  uint32_t tmem_base;
  uint32_t pad_[29];
  float hred[2][4][64];              // NEXT-2: per-warp column sums of the 64 head columns, double buffered
  float qinv_s[kMaxL];               // 1 / |q_j| of the tile the epilogue is working on
};
static_assert(sizeof(TcCtrl) <= kTcCtrlBytes, "control block too large");

__device__ __forceinline__ bool elect_one() {   // one lane of a converged warp: lets the compiler keep the issuing code warp-uniform
  uint32_t pred;
  asm volatile("{\n.reg .pred p;\nelect.sync _|p, 0xffffffff;\nselp.b32 %0, 1, 0, p;\n}" : "=r"(pred));
  return pred != 0;
}
__device__ __forceinline__ uint4 lds128(uint32_t addr) {
  uint4 v;
  asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
  return v;
}
__device__ __forceinline__ float lds32(uint32_t addr) { float v; asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr)); return v; }
__device__ __forceinline__ void sts32(uint32_t addr, float v) { asm volatile("st.shared.f32 [%0], %1;" ::"r"(addr), "f"(v) : "memory"); }

// one token row's half K-slice (4 x 16 bytes): sum of squares
__device__ __forceinline__ void tc_sq4(const uint4 (&x)[4], uint64_t& a, uint64_t& b) {
#pragma unroll
  for (int u = 0; u < 4; ++u) {
    fma_sq_f32x2(a, bf16x2_to_f32x2(x[u].x)); fma_sq_f32x2(b, bf16x2_to_f32x2(x[u].y));
    fma_sq_f32x2(a, bf16x2_to_f32x2(x[u].z)); fma_sq_f32x2(b, bf16x2_to_f32x2(x[u].w));
  }
}
// the same plus the squared difference to the previous frame's values (bit-identical rows give exactly 0)
__device__ __forceinline__ void tc_sq4_diff(const uint4 (&x)[4], const uint4 (&v)[4], uint64_t& a, uint64_t& b, uint64_t& da, uint64_t& db) {
#pragma unroll
  for (int u = 0; u < 4; ++u) {
    const uint64_t x0 = bf16x2_to_f32x2(x[u].x), x1 = bf16x2_to_f32x2(x[u].y), x2 = bf16x2_to_f32x2(x[u].z), x3 = bf16x2_to_f32x2(x[u].w);
    const uint64_t e0 = sub_f32x2(x0, bf16x2_to_f32x2(v[u].x)), e1 = sub_f32x2(x1, bf16x2_to_f32x2(v[u].y));
    const uint64_t e2 = sub_f32x2(x2, bf16x2_to_f32x2(v[u].z)), e3 = sub_f32x2(x3, bf16x2_to_f32x2(v[u].w));
    fma_sq_f32x2(a, x0); fma_sq_f32x2(b, x1); fma_sq_f32x2(a, x2); fma_sq_f32x2(b, x3);
    fma_sq_f32x2(da, e0); fma_sq_f32x2(db, e1); fma_sq_f32x2(da, e2); fma_sq_f32x2(db, e3);
  }
}

// The statistics warps' sweep over one tile.  Thread = (block row `arow`, half `hh` of the row's eight 16-byte units); the
// hardware 128-byte swizzle puts unit u of row r at unit u ^ (r & 7).  Ring position (xs, xph) is carried across tiles.
struct TcAluCtx {
  uint32_t xring, xslot, xfull0, xempty0, stat;   // shared-space addresses; stat = this lane's accumulator of block 0 in this tile's buffer
  uint32_t s0full;                                // barrier: block 0 of a tile whose first block is a dumped part is complete
  int nx, nk, lane, arow;
  uint32_t hh;
};
__device__ __forceinline__ void tc_alu_load(uint32_t base, uint32_t ro, uint32_t uoff, uint32_t swz, uint4 (&x)[4]) {
#pragma unroll
  for (int u = 0; u < 4; ++u) x[u] = lds128(base + ro + (((uoff + (uint32_t)u) ^ swz) << 4));
}
// makes the following instructions wait for the loads into `x` (a data dependency the scoreboard honours)
template <int KW>
__device__ __forceinline__ void tc_alu_fence_loads(const uint4 (&x)[KW][4]) {
  uint32_t acc = 0;
#pragma unroll
  for (int j = 0; j < KW; ++j)
#pragma unroll
    for (int u = 0; u < 4; ++u) acc |= x[j][u].x ^ x[j][u].w;
  asm volatile("" ::"r"(acc) : "memory");
}
__device__ __forceinline__ void tc_alu_release(const TcAluCtx& c, uint32_t& xs, uint32_t& xph) {
  __syncwarp();
  if (c.lane == 0) mbar_arrive(c.xempty0 + xs * 8u);
  if (++xs == (uint32_t)c.nx) { xs = 0; xph ^= 1u; }
}
template <int KW>
__device__ __forceinline__ void tc_alu_tile(const TcAluCtx& c, int mode, int n_rows, int n_blocks, int stride, int prev, bool halo,
                                            int k0, int k1, int nk, uint32_t& xs, uint32_t& xph) {
  const uint32_t roff = (uint32_t)c.arow * 128u, sw = (uint32_t)(c.arow & 7);
  const uint32_t uoff = c.hh << 2;
  const int prow = c.arow - prev;                                        // mode 2: the previous frame's row in the same chunk
  const uint32_t proff = (uint32_t)prow * 128u, psw = (uint32_t)(prow & 7);
  const bool inchunk = mode == 2 && prow >= 0;
  const int hcap = mode == 0 ? stride : 128;
  for (int kc = tc_k_lo(n_blocks, k0); kc < tc_k_hi(n_blocks, k1, nk); kc += KW) {
    const int bf = tc_b_first(kc, k1, n_blocks), be = tc_b_end(kc, k0, n_blocks);
    if (bf >= be) continue;
    uint4 pv[KW][4];                  // this thread's K-slices of the previous frame's row (mode 1: carried from block to block)
    bool have_prev = false;
    if (mode == 1 && (halo || bf)) {  // frame t0 - 1, or frame t0 itself once block 0 has left
      mbar_wait(c.xfull0 + xs * 8u, xph);
      if (c.arow < n_rows) {
        const uint32_t slice = (uint32_t)((n_rows + 7) >> 3) * 1024u;
#pragma unroll
        for (int j = 0; j < KW; ++j) tc_alu_load(c.xring + xs * c.xslot + (uint32_t)j * slice, roff, uoff, sw, pv[j]);
      }
      have_prev = true;
      tc_alu_fence_loads(pv);
      tc_alu_release(c, xs, xph);
    }
    // one block's chunk: `x` receives this thread's K-slices of the row, `pv` holds those of the previous frame's row
    auto step = [&](int b, uint4 (&x)[KW][4], uint4 (&pv)[KW][4]) __attribute__((always_inline)) {
      const int hb = mode == 1 ? n_rows : min(hcap, n_rows - b * stride);
      const uint32_t slice = (uint32_t)((hb + 7) >> 3) * 1024u;
      const bool act = c.arow < hb;
      uint64_t n2a = 0, n2b = 0, Da = 0, Db = 0;     // packed fp32 pairs, all zero bits = (0.f, 0.f)
      mbar_wait(c.xfull0 + xs * 8u, xph);
      if (act) {
#pragma unroll
        for (int j = 0; j < KW; ++j) {
          const uint32_t base = c.xring + xs * c.xslot + (uint32_t)j * slice;
          tc_alu_load(base, roff, uoff, sw, x[j]);
          if (inchunk) tc_alu_load(base, proff, uoff, psw, pv[j]);
        }
      }
      if (act) {
        const bool diff = inchunk || (mode == 1 && have_prev);
#pragma unroll
        for (int j = 0; j < KW; ++j) {
          if (diff) tc_sq4_diff(x[j], pv[j], n2a, n2b, Da, Db); else tc_sq4(x[j], n2a, n2b);
        }
      }
      have_prev = true;
      tc_alu_release(c, xs, xph);   // after the arithmetic: every byte of the slot has arrived in registers by now (an arrive issued
                                    // right behind the loads could complete before them and let the TMA unit overwrite the slot)
      // the chunk's partial sums of a row (two lanes) join block b's accumulators in shared memory
      float n2 = sum_f32x2(n2a) + sum_f32x2(n2b), D = sum_f32x2(Da) + sum_f32x2(Db);
      n2 += __shfl_xor_sync(0xffffffffu, n2, 1);
      D += __shfl_xor_sync(0xffffffffu, D, 1);
      if (act) {   // lane pair (row): the even lane keeps sum x^2, the odd lane sum (x - x_prev)^2
        const float mine = c.hh ? D : n2;
        const uint32_t a = c.stat + (uint32_t)b * 1024u;
        sts32(a, kc == (b == n_blocks - 1 ? k0 : 0) ? mine : lds32(a) + mine);
      }
    };
    uint4 xb[KW][4];
    if (mode == 1) {   // frame walk: the two register sets alternate between "this frame" and "previous frame" (no copies)
      for (int b = bf; b < be; b += 2) {
        step(b, xb, pv);
        if (b + 1 < be) step(b + 1, pv, xb);
      }
    } else {
      for (int b = bf; b < be; ++b) step(b, xb, pv);
    }
    if (n_blocks > 1 && k1 < nk && kc + KW == k1) {   // block 0 has left the sweep: its row sums are complete (the epilogue dumps them early)
      __syncwarp();
      if (c.lane == 0) mbar_arrive(c.s0full);
    }
  }
}

// One block of a tile's epilogue, by four warps that cover the four TMEM lane quarters (q = warp % 4, r = the thread's block row).
// `bar_id`: a named barrier of their own.
__device__ __forceinline__ void tc_epi_block(const TcParams& p, TcCtrl* ctrl, const float* stat, uint32_t tmem_base, const TcTile& tile, int b,
                                             uint32_t ts0, uint32_t tp0, int buf, int it, int q, int lane, uint32_t bar_id, uint32_t& hcnt) {
  const int r = q * 32 + lane;
  const int nk = p.n_kchunks;
  const uint32_t ns = (uint32_t)p.ns;
  const bool rider = p.sig != nullptr || p.heads_part != nullptr;
  const int nqu = (tile.L + 15) >> 4;
  const float inv_d = 1.0f / (float)p.d;
  const float2* st2 = reinterpret_cast<const float2*>(stat) + (size_t)buf * kTcMaxBlocks * 128;
  const bool dump0 = tile.k1 < nk;                               // K-split: block 0 is a part that hands its partial sums to the block's owner
  const float* qinv = ctrl->qinv_s;
  const size_t xslot_f = (size_t)p.xchg_cols * 128;              // floats per exchange slot
  uint32_t ts = ts0 + (uint32_t)b, tp = tp0;
  if (ts >= ns) { ts -= ns; tp ^= 1u; }
  const uint32_t tcol = tmem_base + ts * (uint32_t)p.wslot + ((uint32_t)(q * 32) << 16);
  mbar_wait(smem_u32(&ctrl->tfull[ts]), tp);
  tc_fence_after();
  const int n_wait = b == tile.n_blocks - 1 ? tile.n_wait : 0;   // > 0: this CTA owns a split last block
  if (dump0 && b == 0) {   // accumulator columns (column-major: lanes = rows, coalesced), then the two row sums, then the flag
    float* xo = p.xchg + (size_t)blockIdx.x * xslot_f + r;
    const int ncb = nqu + (rider ? 4 : 0);
    for (int cb = 0; cb < ncb; ++cb) {
      uint32_t v[16];
      tc_ld16(tcol + (uint32_t)cb * 16u, v);
      tc_wait_ld();
#pragma unroll
      for (int j = 0; j < 16; ++j) xo[(size_t)(cb * 16 + j) * 128] = __uint_as_float(v[j]);
    }
    tc_fence_before();
    __syncwarp();
    if (lane == 0) mbar_arrive(smem_u32(&ctrl->tempty[ts]));
    if (tile.n_blocks > 1) mbar_wait(smem_u32(&ctrl->s0full), 0u);   // (complete long before the tile's other blocks)
    else mbar_wait(smem_u32(&ctrl->sfull[buf]), (uint32_t)(it >> 1) & 1u);
    const float2 nd = st2[b * 128 + r];
    xo[(size_t)(p.xchg_cols - 2) * 128] = nd.x;
    xo[(size_t)(p.xchg_cols - 1) * 128] = nd.y;
    __threadfence();
    asm volatile("bar.sync %0, 128;" ::"r"(bar_id) : "memory");       // the four epilogue warps
    if (q == 0 && lane == 0) asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p.xflag + blockIdx.x), "r"(1u) : "memory");
    return;
  }
  if (n_wait > 0) {   // owner of a split block: the other parts were the first thing the CTAs that follow this one swept
    if (lane == 0)
      for (int i = 0; i < n_wait; ++i) {
        unsigned int f;
        do { asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(f) : "l"(p.xflag + tile.peer + i) : "memory"); } while (f == 0u);
      }
    __syncwarp();
  }
  const float* xi = p.xchg + (size_t)tile.peer * xslot_f + r;      // owner: the parts' slots follow one another
  // 16 accumulator columns of this thread's row, the foreign parts added in slot order (a fixed order: bit-reproducible)
  auto ld16 = [&](int cbi, float (&f)[16]) {
    uint32_t v[16];
    tc_ld16(tcol + (uint32_t)cbi * 16u, v);
    tc_wait_ld();
#pragma unroll
    for (int j = 0; j < 16; ++j) f[j] = __uint_as_float(v[j]);
    for (int i = 0; i < n_wait; ++i)
#pragma unroll
      for (int j = 0; j < 16; ++j) f[j] += xi[(size_t)i * xslot_f + (size_t)(cbi * 16 + j) * 128];
  };
  const int hb = tc_block_rows(tile, b);
  const int out_lo = tile.mode == 2 ? (b == 0 ? tile.halo : tile.prev) : 0;
  const bool valid = r < hb && r >= out_lo;
  const int64_t row = (int64_t)tile.row0 + (int64_t)b * tile.stride + r;
  float m = -INFINITY;
  if (n_wait == 0) {   // the common case: two column groups in flight per wait
    for (int cb = 0; cb < nqu; cb += 2) {
      uint32_t v0[16], v1[16];
      tc_ld16(tcol + (uint32_t)cb * 16u, v0);
      if (cb + 1 < nqu) tc_ld16(tcol + (uint32_t)(cb + 1) * 16u, v1);
      tc_wait_ld();
#pragma unroll
      for (int j = 0; j < 16; ++j) {
        const int col = cb * 16 + j;
        if (col < tile.L) m = fmaxf(m, __uint_as_float(v0[j]) * qinv[col]);
      }
      if (cb + 1 < nqu) {
#pragma unroll
        for (int j = 0; j < 16; ++j) {
          const int col = cb * 16 + 16 + j;
          if (col < tile.L) m = fmaxf(m, __uint_as_float(v1[j]) * qinv[col]);
        }
      }
    }
  } else {
    for (int cb = 0; cb < nqu; ++cb) {
      float v[16];
      ld16(cb, v);
#pragma unroll
      for (int j = 0; j < 16; ++j) {
        const int col = cb * 16 + j;
        if (col < tile.L) m = fmaxf(m, v[j] * qinv[col]);
      }
    }
  }
  if (p.heads_part != nullptr) {   // NEXT-2: column 0 -> the learned spatial map, all 64 -> per-block column sums (fixed order)
    float tot[2];
#pragma unroll
    for (int grp = 0; grp < 2; ++grp) {
      float x[32];
#pragma unroll
      for (int cb = 0; cb < 2; ++cb) {
        float v[16];
        ld16(nqu + grp * 2 + cb, v);
#pragma unroll
        for (int j = 0; j < 16; ++j) x[cb * 16 + j] = valid ? v[j] : 0.f;
      }
      if (grp == 0) {
        float below = 0.f;
        if (valid) {
          const float M = sigmoidf_acc(x[0] + p.heads_bias);
          p.heads_m[row] = M;
          below = M < p.heads_tau ? 1.f : 0.f;
        }
        x[0] = below;
      }
      // transpose-reduce over the warp: 31 shuffles leave the total of column `lane` in lane `lane`
#pragma unroll
      for (int w = 16; w >= 1; w >>= 1) {
        const bool up = (lane & w) != 0;
#pragma unroll
        for (int i = 0; i < w; ++i) {
          const float send = up ? x[i] : x[i + w], keep = up ? x[i + w] : x[i];
          x[i] = keep + __shfl_xor_sync(0xffffffffu, send, w);
        }
      }
      tot[grp] = x[0];
    }
    const int hbuf = (int)(hcnt++ & 1u);
    ctrl->hred[hbuf][q][lane] = tot[0];
    ctrl->hred[hbuf][q][32 + lane] = tot[1];
    asm volatile("bar.sync %0, 128;" ::"r"(bar_id) : "memory");       // the four epilogue warps
    if (r < 64)
      p.heads_part[((int64_t)tile.part0 + b) * 64 + r] = (ctrl->hred[hbuf][0][r] + ctrl->hred[hbuf][1][r]) + (ctrl->hred[hbuf][2][r] + ctrl->hred[hbuf][3][r]);
  } else if (rider) {   // NEXT-1: the 64 accumulator columns after the query columns are r_k . x: their signs are the hash bits
    unsigned long long bits = 0ull;
#pragma unroll
    for (int cb = 0; cb < 4; ++cb) {
      float v[16];
      ld16(nqu + cb, v);
#pragma unroll
      for (int j = 0; j < 16; ++j) bits |= (unsigned long long)(v[j] >= 0.f) << (cb * 16 + j);
    }
    if (valid) p.sig[row] = bits;
  }
  tc_fence_before();
  __syncwarp();
  if (lane == 0) mbar_arrive(smem_u32(&ctrl->tempty[ts]));
  mbar_wait(smem_u32(&ctrl->sfull[buf]), (uint32_t)(it >> 1) & 1u);   // (true at once after the tile's first wait)
  float2 nd = st2[b * 128 + r];
  for (int i = 0; i < n_wait; ++i) {
    nd.x += xi[(size_t)i * xslot_f + (size_t)(p.xchg_cols - 2) * 128];
    nd.y += xi[(size_t)i * xslot_f + (size_t)(p.xchg_cols - 1) * 128];
  }
  if (valid) {
    p.s[row] = sqrtf(nd.x * inv_d);
    p.dnorm[row] = sqrtf(nd.y);
    p.rel[row] = nd.x > 0.f ? m / sqrtf(nd.x) : 0.f;
  }
  if (n_wait > 0) {   // every warp has read the slots: re-arm their flags for the next launch
    asm volatile("bar.sync %0, 128;" ::"r"(bar_id) : "memory");
    if (q == 0 && lane < n_wait) p.xflag[tile.peer + lane] = 0u;
  }
}

template <int KW, bool HELP>   // 64-column K-slices per chunk; the statistics warps join the epilogue of the CTA's last tile
__global__ void __launch_bounds__(kTcThreads, 1)
k_score_tc(const __grid_constant__ TcMaps maps, const __grid_constant__ TcParams p) {
  extern __shared__ unsigned char smem_raw[];
  unsigned char* smem = reinterpret_cast<unsigned char*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  TcCtrl* ctrl = reinterpret_cast<TcCtrl*>(smem);
  float* stat = reinterpret_cast<float*>(smem + kTcCtrlBytes);
  const uint32_t sbase = smem_u32(smem);
  const uint32_t qring = sbase + kTcCtrlBytes + kTcStatBytes;
  const uint32_t xring = qring + (uint32_t)p.nq * (uint32_t)p.qslot_bytes;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  // roles: warps 0-3 epilogue (TMEM lane quarter = warp % 4), 4-11 statistics, 12 TMA producer, 13 MMA issuer (+ TMEM allocation):
  // two statistics warps and one epilogue warp on every scheduler partition
  const int tile_lo = p.cta_off[blockIdx.x], tile_hi = p.cta_off[blockIdx.x + 1];
  const int nk = p.n_kchunks;
  const int nx = p.nx;
  constexpr int kw = KW;
  const uint32_t xslot = (uint32_t)kw * (uint32_t)kTcSliceBytes;
  const bool rider = p.sig != nullptr || p.heads_part != nullptr;   // 64 more B rows after the query rows (hash rows or head weights)
  const uint32_t ns = (uint32_t)p.ns;                    // accumulator slots, used round-robin block after block
  const uint32_t xfull0 = smem_u32(&ctrl->xfull[0]), xempty0 = smem_u32(&ctrl->xempty[0]);
  const uint32_t qfull0 = smem_u32(&ctrl->qfull[0]), qempty0 = smem_u32(&ctrl->qempty[0]);
  const uint32_t tfull0 = smem_u32(&ctrl->tfull[0]), tempty0 = smem_u32(&ctrl->tempty[0]);

  pdl_launch_dependents();   // the segment kernel may be scheduled as SMs free up; it waits for this grid to complete
  if (warp == kTcWarpMma && lane == 0) {
    for (int i = 0; i < kTcMaxXSlots; ++i) { mbar_init(xfull0 + 8u * i, 1); mbar_init(xempty0 + 8u * i, 1 + kTcAluWarps); }
    for (int i = 0; i < 4; ++i) { mbar_init(qfull0 + 8u * i, 1); mbar_init(qempty0 + 8u * i, 1); }
    for (int i = 0; i < 2; ++i) {
      mbar_init(smem_u32(&ctrl->sfull[i]), kTcAluWarps); mbar_init(smem_u32(&ctrl->sempty[i]), 4);
    }
    for (int i = 0; i < kTcMaxBlocks; ++i) { mbar_init(tfull0 + 8u * i, 1); mbar_init(tempty0 + 8u * i, 4); }
    mbar_init(smem_u32(&ctrl->s0full), kTcAluWarps);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == kTcWarpMma) {   // TMEM: all 512 columns (one CTA per SM): 4 to 10 accumulator slots of pad16(L) columns
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&ctrl->tmem_base)), "r"(512) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  if (warp == kTcWarpTma && lane == 0) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(&maps.x[15]) : "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(&maps.q[0]) : "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(&maps.q[2]) : "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = ctrl->tmem_base;
  pdl_wait();   // plain (non-cooperative) launches are chained behind k_qprep: the set-up above overlaps its tail

  if (warp == kTcWarpTma) {
    // ===================================================================== TMA producer (the whole warp walks the list, one lane issues)
    uint32_t xs = 0, xph = 0, qs = 0, qph = 0;
    uint64_t pol_stream, pol_keep;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol_stream));
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol_keep));
    for (int t = tile_lo; t < tile_hi; ++t) {
      const TcTile tile = p.tiles[t];
      const int nqu = (tile.L + 15) >> 4;
      const uint32_t qbytes = (uint32_t)(nqu + (rider ? 4 : 0)) * 2048u * (uint32_t)kw;
      for (int kc = tc_k_lo(tile.n_blocks, tile.k0); kc < tc_k_hi(tile.n_blocks, tile.k1, nk); kc += kw) {
        const int bf = tc_b_first(kc, tile.k1, tile.n_blocks), be = tc_b_end(kc, tile.k0, tile.n_blocks);
        if (bf >= be) continue;
        // frame walk: the chunk of the frame before the first block taking part rides along for the statistics warps only (block -1 =
        // frame t0 - 1, the halo; block 0 itself once it has left)
        const int b_lo = tile.mode == 1 ? (bf ? 0 : (tile.halo ? -1 : 0)) : bf;
        {   // the request's query rows of these K-slices (+ the rider rows): one B tile per slice
          mbar_wait(qempty0 + 8u * qs, qph ^ 1u);
          if (elect_one()) {
            const uint32_t bar = qfull0 + 8u * qs;
            mbar_expect_tx(bar, qbytes);
            uint32_t sq = qring + qs * (uint32_t)p.qslot_bytes;
            for (int j = 0; j < kw; ++j) {
              int qr = tile.q_row0;
              for (int i = 0; i < (nqu >> 2); ++i) { tma_load_3d_hint(sq, &maps.q[0], bar, 0, qr, kc + j, pol_keep); sq += 8192; qr += 64; }
              if (nqu & 2) { tma_load_3d_hint(sq, &maps.q[1], bar, 0, qr, kc + j, pol_keep); sq += 4096; qr += 32; }
              if (nqu & 1) { tma_load_3d_hint(sq, &maps.q[2], bar, 0, qr, kc + j, pol_keep); sq += 2048; }
              if (rider) { tma_load_3d_hint(sq, &maps.r, bar, 0, 0, kc + j, pol_keep); sq += 8192; }
            }
          }
          if (++qs == (uint32_t)p.nq) { qs = 0; qph ^= 1u; }
        }
        for (int b = b_lo; b < be; ++b) {
          const int h = b < 0 ? tile.n_rows : tc_block_rows(tile, b);
          const int h8 = (h + 7) >> 3;                               // box height in 8-row swizzle atoms
          mbar_wait(xempty0 + 8u * xs, xph ^ 1u);
          if (elect_one()) {
            const uint32_t bar = xfull0 + 8u * xs;
            mbar_expect_tx(bar, (uint32_t)h8 * 1024u * (uint32_t)kw);
            // one box = kw slices of h8 * 8 rows, slice after slice; rows past the end of X are zero-filled by the TMA unit,
            // rows past the block are never used
            // a video tile's halo and last frame are read by two CTAs (as halo and as a block), and so is the frame before a
            // split last frame: ordinary priority; the rest of X is read once: evict first
            if (tile.mode == 1 && (b < bf || b == tile.n_blocks - 1 || (b == tile.n_blocks - 2 && tile.k0 > 0))) tma_load_3d(xring + xs * xslot, &maps.x[h8 - 1], bar, 0, tile.row0 + b * tile.stride, kc);
            else tma_load_3d_hint(xring + xs * xslot, &maps.x[h8 - 1], bar, 0, tile.row0 + b * tile.stride, kc, pol_stream);
          }
          if (++xs == (uint32_t)nx) { xs = 0; xph ^= 1u; }
        }
      }
    }
  } else if (warp == kTcWarpMma) {
    // ===================================================================== MMA issuer (the whole warp walks the list, one lane issues)
    uint32_t xs = 0, xph = 0, qs = 0, qph = 0, ts0 = 0, tp0 = 0;   // ts0 / tp0: accumulator slot and phase of the tile's block 0
    for (int t = tile_lo; t < tile_hi; ++t) {
      const TcTile tile = p.tiles[t];
      const int nqb = ((tile.L + 15) >> 4) + (rider ? 4 : 0);
      const uint32_t idesc = umma_idesc_bf16(nqb << 4);   // N = pad16(L) (+ 64 rider rows)
      const bool early0 = tile.n_blocks > 1 && tile.k1 < nk;   // the first block is a dumped part that leaves the sweep at k1
      for (int kc = tc_k_lo(tile.n_blocks, tile.k0); kc < tc_k_hi(tile.n_blocks, tile.k1, nk); kc += kw) {
        const int bf = tc_b_first(kc, tile.k1, tile.n_blocks), be = tc_b_end(kc, tile.k0, tile.n_blocks);
        if (bf >= be) continue;
        const bool halo = tile.mode == 1 && (tile.halo || bf);
        mbar_wait(qfull0 + 8u * qs, qph);
        tc_fence_after();
        const uint32_t qbase = qring + qs * (uint32_t)p.qslot_bytes;
        if (halo) {   // not an MMA operand: release our share of the slot, behind the MMAs issued so far (which keeps the order) and
                      // not before the chunk has landed (an arrival ahead of the slot's previous phase would be counted there)
          mbar_wait(xfull0 + 8u * xs, xph);
          if (elect_one()) tc_commit(xempty0 + 8u * xs);
          if (++xs == (uint32_t)nx) { xs = 0; xph ^= 1u; }
        }
        for (int b = bf; b < be; ++b) {
          uint32_t ts = ts0 + (uint32_t)b, tp = tp0;
          if (ts >= ns) { ts -= ns; tp ^= 1u; }
          const int kstart = b == tile.n_blocks - 1 ? tile.k0 : 0;   // the block's first K-chunk
          if (kc == kstart) {   // the accumulator slot must have been drained by the epilogue of its previous use
            mbar_wait(tempty0 + 8u * ts, tp ^ 1u);
            tc_fence_after();
          }
          mbar_wait(xfull0 + 8u * xs, xph);
          tc_fence_after();
          const uint32_t slice = (uint32_t)((tc_block_rows(tile, b) + 7) >> 3) * 1024u;   // bytes between the K-slices of this chunk
          const uint32_t xbase = xring + xs * xslot;
          const uint32_t d_tmem = tmem_base + ts * (uint32_t)p.wslot;
          if (elect_one()) {
            for (int j = 0; j < kw; ++j) {
              // M = 128: rows past the block read whatever follows in the slot (their accumulator rows are never used)
              const uint64_t adesc = umma_desc_sw128(xbase + (uint32_t)j * slice);
              const uint64_t bdesc = umma_desc_sw128(qbase + (uint32_t)j * (uint32_t)nqb * 2048u);
#pragma unroll
              for (int k = 0; k < 4; ++k)   // 4 x K=16 inside the 128-byte swizzle atom: +32 B = +2 in the 16-byte address field
                tc_mma_bf16(d_tmem, adesc + (uint64_t)(2 * k), bdesc + (uint64_t)(2 * k), idesc, (uint32_t)((kc - kstart) | j | k));
            }
            tc_commit(xempty0 + 8u * xs);
          }
          if (++xs == (uint32_t)nx) { xs = 0; xph ^= 1u; }
        }
        if (elect_one()) {
          tc_commit(qempty0 + 8u * qs);
          if (early0 && kc + kw == tile.k1) tc_commit(tfull0 + 8u * ts0);   // block 0 has left the sweep: the epilogue may dump it now
        }
        if (++qs == (uint32_t)p.nq) { qs = 0; qph ^= 1u; }
      }
      if (elect_one())
        for (int b = early0 ? 1 : 0; b < tile.n_blocks; ++b) { const uint32_t ts = ts0 + (uint32_t)b; tc_commit(tfull0 + 8u * (ts >= ns ? ts - ns : ts)); }
      ts0 += (uint32_t)tile.n_blocks;
      if (ts0 >= ns) { ts0 -= ns; tp0 ^= 1u; }
    }
  } else {
    // ===================================================================== epilogue warps (0-3) and statistics warps (4-11)
    // Both end in the same tile-epilogue loop below (one copy of its code): the epilogue warps run it over all tiles, the
    // statistics warps (HELP) join it for the CTA's last tile, whose epilogue nothing hides, with two blocks in three.
    const bool epi = warp < 4;
    const int q = warp & 3;                  // TMEM lane quarter this warp may access (warp % 4)
    const int r = q * 32 + lane;             // block row
    uint32_t ts0 = 0, tp0 = 0, hcnt = 0;
    int it = 0, t_first = tile_lo, b_first = 0;
    uint32_t bar_id = 1;                     // named barrier of this group of four warps
    bool q_ok = p.Q == nullptr;
    if (epi) {
      // a0 inside the same launch: while the first chunks stream in, these four warps compute 1 / |q_j| for this CTA's
      // share of the query rows (row j belongs to CTA j % gridDim.x).  Every CTA of the grid is co-resident (cooperative
      // launch), so the first epilogue may wait on the grid-wide counter for the other CTAs' shares.
      if (p.Q != nullptr) {
        const uint4* Qv = static_cast<const uint4*>(p.Q);
        const int n16 = p.d >> 3;              // 16-byte pieces per bf16 row
        for (long long j = (long long)blockIdx.x + (long long)q * gridDim.x; j < p.nQ; j += 4ll * gridDim.x) {
          float acc = 0.f;
          for (int i = lane; i < n16; i += 32) {
            const uint4 v = ld_nc16(Qv + j * n16 + i);
            const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
            for (int k = 0; k < 4; ++k) { const float a0 = bf_lo(w[k]), a1 = bf_hi(w[k]); acc = fmaf(a0, a0, acc); acc = fmaf(a1, a1, acc); }
          }
          acc = warp_sum(acc);
          if (lane == 0) p.qinv[j] = acc > 0.f ? 1.0f / sqrtf(acc) : 0.f;
        }
        __threadfence();
        asm volatile("bar.sync 1, 128;" ::: "memory");       // the four epilogue warps
        if (q == 0 && lane == 0) atomicAdd(p.q_ready, 1ull);
      }
    } else {
      // CUDA-core statistics: two threads per block row
      TcAluCtx c;
      c.xring = xring; c.xslot = xslot; c.xfull0 = xfull0; c.xempty0 = xempty0; c.s0full = smem_u32(&ctrl->s0full);
      c.nx = nx; c.nk = nk; c.lane = lane;
      c.arow = ((warp - 4) << 4) + (lane >> 1);
      c.hh = (uint32_t)lane & 1u;
      uint32_t xs = 0, xph = 0, nbsum = 0;
      int ia = 0;
      for (int t = tile_lo; t < tile_hi; ++t, ++ia) {
        const TcTile tile = p.tiles[t];
        const int buf = ia & 1;
        c.stat = smem_u32(stat) + (uint32_t)buf * (kTcMaxBlocks * 1024u) + (uint32_t)(c.arow * 2 + (int)c.hh) * 4u;   // + b * 1024: block b
        mbar_wait(smem_u32(&ctrl->sempty[buf]), ((uint32_t)(ia >> 1) & 1u) ^ 1u);
        tc_alu_tile<KW>(c, tile.mode, tile.n_rows, tile.n_blocks, tile.stride, tile.prev, tile.mode == 1 && tile.halo != 0, tile.k0, tile.k1, nk, xs, xph);
        __syncwarp();
        if (lane == 0) mbar_arrive(smem_u32(&ctrl->sfull[buf]));
        if (HELP && t + 1 < tile_hi) nbsum += (uint32_t)tile.n_blocks;   // accumulator slots are handed out round-robin, block after block
      }
      t_first = tile_hi;
      if (HELP && tile_hi > tile_lo) {   // join the last tile's epilogue: warps 4-7 blocks b % 3 == 1, warps 8-11 b % 3 == 2
        t_first = tile_hi - 1;
        it = t_first - tile_lo;
        ts0 = nbsum % ns; tp0 = (nbsum / ns) & 1u;
        b_first = warp < 8 ? 1 : 2;
        bar_id = (uint32_t)(1 + b_first);
        asm volatile("bar.sync 4, 384;" ::: "memory");     // the epilogue warps have staged the tile's 1 / |q_j|
      }
    }
    for (int t = t_first; t < tile_hi; ++t, ++it) {
      const TcTile tile = p.tiles[t];
      const int buf = it & 1;
      const bool helped = HELP && t == tile_hi - 1;
      if (epi) {
        if (!(tile.k1 < nk && tile.n_blocks == 1)) {   // the tile's 1 / |q_j| into shared memory: the column loop below reads them as broadcasts
          if (!q_ok) {   // all CTAs' shares of qinv are written (first tile only; normally long since true)
            unsigned long long seen;
            do { asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(seen) : "l"(p.q_ready) : "memory"); } while (seen < (unsigned long long)gridDim.x);
            q_ok = true;
          }
          asm volatile("bar.sync 1, 128;" ::: "memory");       // the four epilogue warps are done with the previous tile's values
          if (r < tile.L) ctrl->qinv_s[r] = p.qinv[tile.q_row0 + r];
          asm volatile("bar.sync 1, 128;" ::: "memory");
        }
        if (helped) asm volatile("bar.arrive 4, 384;" ::: "memory");   // qinv_s is staged
      }
      for (int b = b_first; b < tile.n_blocks; b += helped ? 3 : 1)
        tc_epi_block(p, ctrl, stat, tmem_base, tile, b, ts0, tp0, buf, it, q, lane, bar_id, hcnt);
      if (epi) {
        __syncwarp();
        if (lane == 0) mbar_arrive(smem_u32(&ctrl->sempty[buf]));
      }
      ts0 += (uint32_t)tile.n_blocks;
      if (ts0 >= ns) { ts0 -= ns; tp0 ^= 1u; }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (tid == 0 && p.Q != nullptr) {   // every CTA is past its wait on q_ready[0] by now; the last one out zeroes both counters
    __threadfence();
    if (atomicAdd(p.q_ready + 1, 1ull) == (unsigned long long)gridDim.x - 1ull) { p.q_ready[0] = 0ull; p.q_ready[1] = 0ull; __threadfence(); }
  }
  if (warp == kTcWarpMma) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(512) : "memory");
  }
}

// ------------------------------------------------------------------------------------------------ host side
// Schedule.  The rows of the batch are laid out as STRIPS (a single-frame segment; the patch rows of one group of
// consecutive frames of a video; a short-frame segment), each strip row costing the rows it streams (frames of the group
// + half a row for the L2-served halo).  CTAs take consecutive, equal-cost runs of strip rows, cut at single-row
// granularity (TMA boxes are rounded up to 8 rows; the few rows read twice are L2 hits); a run is cut into tiles of at
// most 8 blocks, each tile paying a fixed cost for the query rows it streams.  Consecutive CTAs sweep neighbouring rows
// of the same frames at the same time, so the halo chunks are L2 hits.
struct TcCost {
  // Roughly microseconds of one CTA with the whole machine streaming (fitted to per-CTA sweep times on the five workloads,
  // profiles/r02_schedule.md).  A block costs almost the same whatever its height (M = 128 MMAs read 128 rows of shared memory, every
  // chunk is a barrier round trip and a dependent chain in the statistics warps); a frame-walk block differences every row, a window
  // of a short-frame segment also reads every row twice.  A tile pays for the query rows it streams and for its halo chunks (by its
  // share of K), a constant for the refill of the pipeline, and for the accumulator slots it has to wait for: the epilogue of the
  // tile before it drains one slot in about t_epi.
  double c_blk = 14.0, w_row = 0.025;
  double f_walk = 1.28, f_short = 1.7;
  double w_halo = 0.077;   // per row of a halo chunk
  double w_q = 0.055;      // per (padded) query row
  double c_tile = 1.5;
  double epi0 = 0.35, epi_col = 0.013;   // t_epi = epi0 + epi_col * accumulator columns
};

inline size_t tc_max_tiles(const mas_segment* segs, int32_t n_segs) {
  size_t tiles = 0;
  for (int32_t k = 0; k < n_segs; ++k) tiles += (size_t)(((int64_t)segs[k].n_frames * segs[k].n_patches) / 64) + (size_t)segs[k].n_frames + 4;
  return tiles + 2048;
}
inline size_t tc_max_parts(const mas_segment* segs, int32_t n_segs) {   // blocks of all tiles (NEXT-2 partial slots)
  size_t blocks = 0;
  for (int32_t k = 0; k < n_segs; ++k) blocks += (size_t)(((int64_t)segs[k].n_frames * segs[k].n_patches) / 32) + 2 * (size_t)segs[k].n_frames + 8;
  return blocks + 8 * 2048;
}
inline size_t tc_xchg_bytes() { return (size_t)kTcMaxCtas * (kMaxL + 2) * 128 * sizeof(float); }   // K-split exchange slots, worst case
inline size_t tc_schedule_bytes(const mas_segment* segs, int32_t n_segs) {
  return tc_max_tiles(segs, n_segs) * sizeof(TcTile) + 1024 * sizeof(int32_t) + 256;
}

// Builds the tile list (grouped per CTA) and the per-CTA offsets into `h_dst`; `d_dst` is where the image will live.
// `rider`: the launch appends 64 B rows (NEXT-1 / NEXT-2), which needs every L <= 64.
// `ksplit`: CTAs may share a row block along K (needs all CTAs co-resident: the owner of a block waits for the other parts).
inline void tc_build_schedule(TcSchedule& sc, const mas_segment* segs, int32_t n_segs, const int64_t* q_off, int32_t d, int32_t dtype,
                              int sm_count, char* h_dst, char* d_dst, bool rider = false, bool ksplit = true) {
  sc = TcSchedule();
  if (dtype != MAS_BF16 || d % 64 != 0 || sm_count < 1 || sm_count > 1000) return;
  const TcCost cw;
  int maxL = 1;
  for (int32_t k = 0; k < n_segs; ++k) maxL = std::max(maxL, (int)(q_off[segs[k].request + 1] - q_off[segs[k].request]));
  const int npad_max = (maxL + 15) / 16 * 16 + (rider ? 64 : 0);
  if (npad_max > 128) return;
  sc.wslot = npad_max;
  sc.xchg_cols = npad_max + 2;
  sc.ns = std::min(kTcMaxBlocks, 512 / npad_max);
  const int NS = sc.ns;
  sc.kw = (d % 128 == 0) ? 2 : 1;
  sc.qslot_bytes = npad_max * 128 * sc.kw;
  {   // shared memory: control + statistics, then the query ring (at least 3 slots where they leave 128 KB for the token ring)
    const int avail = kTcSmemBytes - 1024 - kTcCtrlBytes - kTcStatBytes, xs_bytes = sc.kw * kTcSliceBytes;
    sc.nx = std::min(kTcMaxXSlots, (avail - 2 * sc.qslot_bytes) / xs_bytes);
    sc.nq = (avail - sc.nx * xs_bytes) / sc.qslot_bytes;
    if (sc.nq < 3 && (sc.nx - 1) * xs_bytes >= 128 * 1024) { --sc.nx; sc.nq = (avail - sc.nx * xs_bytes) / sc.qslot_bytes; }
    sc.nq = std::max(2, std::min(4, sc.nq));
    sc.smem_bytes = 1024 + kTcCtrlBytes + kTcStatBytes + sc.nq * sc.qslot_bytes + sc.nx * xs_bytes;
  }

  // The batch as STRIPS of row blocks that may share a tile: the blocks of a single-frame segment (one height, a multiple of 8
  // rows: a TMA box is a whole number of 8-row swizzle atoms, so no row is fetched by two CTAs); one block of patch rows
  // [r0, r0 + R) of a video segment through all its frames (block i = frame i); the overlapping windows of a short-frame segment
  // (window i starts at row i (128 - P) and scores its rows from P on, window 0 all of them).  A tile takes up to NS consecutive
  // blocks of a strip.
  struct Strip { int32_t seg, mode, r0, R, P, stride; int64_t n, nblk; double cb, c_q, c_halo, t_epi; };
  std::vector<Strip> strips;
  for (int32_t k = 0; k < n_segs; ++k) {
    const mas_segment& s = segs[k];
    const int L = (int)(q_off[s.request + 1] - q_off[s.request]);
    const int ncol = (L + 15) / 16 * 16 + (rider ? 64 : 0);
    const double c_q = cw.w_q * ncol;                      // the query rows a tile streams (scaled by its share of K)
    const double t_epi = cw.epi0 + cw.epi_col * ncol;
    const int64_t n = (int64_t)s.n_frames * s.n_patches;
    if (s.n_frames == 1) {
      const int64_t nb = (n + 127) / 128;
      const int stride = (int)(((n + nb - 1) / nb + 7) / 8 * 8);
      strips.push_back(Strip{k, 0, 0, 0, 0, stride, n, nb, cw.c_blk + cw.w_row * ((double)n / nb), c_q, 0.0, t_epi});
    } else if (s.n_patches >= 64) {
      const int nb = (s.n_patches + 127) / 128;            // row blocks of nearly equal height, in whole 8-row swizzle atoms
      for (int j = 0; j < nb; ++j) {
        const int oct = (s.n_patches + 7) / 8;
        const int r0 = 8 * (int)((int64_t)j * oct / nb), r1 = j + 1 == nb ? s.n_patches : 8 * (int)((int64_t)(j + 1) * oct / nb);
        strips.push_back(Strip{k, 1, r0, r1 - r0, s.n_patches, s.n_patches, n, (int64_t)s.n_frames, cw.f_walk * (cw.c_blk + cw.w_row * (r1 - r0)), c_q,
                               cw.w_halo * (r1 - r0), t_epi});
      }
    } else {
      const int64_t sdt = 128 - s.n_patches;
      strips.push_back(Strip{k, 2, 0, 0, s.n_patches, (int32_t)sdt, n, n <= 128 ? 1 : (n - 128 + sdt - 1) / sdt + 1, cw.f_short * (cw.c_blk + cw.w_row * 128.0), c_q, 0.0,
                             t_epi});
    }
  }
  const int S = (d / 64) / sc.kw;                          // K-steps of a full sweep
  const bool can_split = ksplit && S >= 4;
  // Cost of a run of nb consecutive blocks of a strip, cut into the fewest tiles, whose first block is swept for the share `a` of K
  // and whose last block for the share `b` (a one-block run: the share a + b - 1).  `at0`: the run starts with the strip's first
  // block and all of its K (no halo for the first tile).  `prev_nb`, `prev_epi`: blocks and t_epi of the CTA's previous tile.
  auto run_cost = [&](const Strip& st, int64_t nb, double a, double b, bool at0, int prev_nb, double prev_epi) {
    if (nb <= 0) return 0.0;
    const int64_t nt = (nb + NS - 1) / NS;
    const double per = (double)nb / nt;                  // blocks per tile
    const double wait0 = prev_epi * std::max(0.0, prev_nb + per - NS), wait = st.t_epi * std::max(0.0, 2.0 * per - NS);
    if (nb == 1) return (st.cb + st.c_q + (at0 ? 0.0 : st.c_halo)) * (a + b - 1.0) + cw.c_tile + wait0;
    return st.cb * ((double)(nb - 2) + a + b) + (double)nt * (st.c_q + cw.c_tile) + (double)(nt - (at0 ? 1 : 0)) * st.c_halo + wait0 + (double)(nt - 1) * wait;
  };
  double total = 0.0;
  for (const Strip& st : strips) total += run_cost(st, st.nblk, 1.0, 1.0, true, 0, 0.0);
  const int n_ctas = (int)std::min<int64_t>(std::min(sm_count, kTcMaxCtas), std::max<int64_t>(1, (int64_t)(total / 12.0)));

  std::vector<TcTile> tiles;
  std::vector<int> cta_first(n_ctas + 1, 0);
  // blocks [i0, i1) of a strip as one tile: block i1 - 1 from K-step s0 on, block i0 up to K-step s1 (one block: [s0, s1))
  auto emit = [&](const Strip& st, int64_t i0, int64_t i1, int s0, int s1) {
    const mas_segment& s = segs[st.seg];
    TcTile t{};
    t.mode = st.mode; t.seg = st.seg;
    t.q_row0 = (int32_t)q_off[s.request];
    t.L = (int32_t)(q_off[s.request + 1] - q_off[s.request]);
    t.k0 = s0 * sc.kw; t.k1 = s1 * sc.kw; t.peer = -1;
    t.n_blocks = (int32_t)(i1 - i0); t.stride = st.stride;
    if (st.mode == 0) {
      t.row0 = (int32_t)(s.row0 + i0 * st.stride); t.n_rows = (int32_t)(std::min<int64_t>(st.n, i1 * st.stride) - i0 * st.stride);
    } else if (st.mode == 1) {                              // frames [i0, i1) of the strip's row block
      t.row0 = (int32_t)(s.row0 + i0 * s.n_patches + st.r0); t.n_rows = st.R; t.prev = s.n_patches; t.halo = i0 > 0 ? 1 : 0;
    } else {
      t.row0 = (int32_t)(s.row0 + i0 * st.stride); t.n_rows = (int32_t)(std::min<int64_t>(st.n, (i1 - 1) * st.stride + 128) - i0 * st.stride);
      t.prev = st.P; t.halo = i0 > 0 ? st.P : 0;            // leading rows of the first window that are loaded for their successors only
    }
    tiles.push_back(t);
  };
  // One pass with a fixed per-CTA target: CTAs fill up to the target in strip order, first with whole blocks, then with the LAST
  // K-steps of the next block (K-split: that CTA owns the block and sweeps its part at the very end; the CTA that follows starts
  // with the block's remaining K-steps, which are complete and dumped early in its sweep); the last CTA takes what is left.
  // Returns the last CTA's load.
  auto assign = [&](double target, bool commit) {
    int c = 0;
    double load = 0.0;
    int owner = -1;                                     // index of the tile that owns the block being split
    int prev_nb = 0;                                    // the CTA's previous tile
    double prev_epi = 0.0;
    if (commit) { tiles.clear(); std::fill(cta_first.begin(), cta_first.end(), 0); }
    auto close_cta = [&]() {
      if (c + 1 < n_ctas) { load = 0.0; prev_nb = 0; ++c; if (commit) cta_first[c] = (int)tiles.size(); }
    };
    auto took = [&](const Strip& st, int64_t nb) {      // a run of nb blocks joined the CTA: its last tile is the previous one now
      const int64_t nt = (nb + NS - 1) / NS;
      prev_nb = (int)(nb - nb * (nt - 1) / nt); prev_epi = st.t_epi;
    };
    // cost of the run of nb blocks from block i on, `ks` K-steps of block i already handed out (from the top), the last block
    // taking the share b of K
    auto cost = [&](const Strip& st, int64_t i, int ks, int64_t nb, double b) {
      return run_cost(st, nb, (double)(S - ks) / S, b, i == 0 && ks == 0, prev_nb, prev_epi);
    };
    // the run of blocks [i, i + nb): block i up to K-step e0 (a dumped part if e0 < S), the last block from K-step s_last on (the
    // owner's part if s_last > 0), as the fewest tiles
    auto emit_run = [&](const Strip& st, int64_t i, int64_t nb, int e0, int s_last) {
      const int64_t nt = (nb + NS - 1) / NS;
      for (int64_t j = 0; j < nt; ++j) {
        const int64_t b0 = i + nb * j / nt, b1 = i + nb * (j + 1) / nt;
        emit(st, b0, b1, j + 1 == nt ? s_last : 0, j == 0 ? e0 : S);
        const int me = (int)tiles.size() - 1;
        if (j == 0 && e0 < S) {                         // a dumping part: slot c, read by the owner
          tiles[owner].n_wait += 1;
          if (tiles[owner].peer < 0) tiles[owner].peer = c;
        }
        if (j + 1 == nt && s_last > 0 && !(nb == 1 && e0 < S)) owner = me;
      }
    };
    for (const Strip& st : strips) {
      int64_t i = 0;
      int ks = 0;                                       // K-steps of block i already handed out
      while (i < st.nblk) {
        const int64_t m_all = st.nblk - i;
        if (c + 1 >= n_ctas || load + cost(st, i, ks, m_all, 1.0) <= target) {   // the rest of the strip
          if (commit) emit_run(st, i, m_all, S - ks, 0);
          load += cost(st, i, ks, m_all, 1.0);
          took(st, m_all);
          break;
        }
        int64_t lo = 0, hi = m_all - 1;                 // whole blocks that fit
        while (lo < hi) { const int64_t mid = (lo + hi + 1) / 2; if (load + cost(st, i, ks, mid, 1.0) <= target) lo = mid; else hi = mid - 1; }
        int64_t nb = lo;
        int fit = 0;                                    // K-steps of block i + nb on top
        if (can_split) {
          const double b_none = nb == 0 ? (double)ks / S : 0.0;                          // (a one-block run's share is a + b - 1)
          const double base = cost(st, i, ks, nb + 1, b_none);                           // with none of the K-steps of block i + nb
          const double per = cost(st, i, ks, nb + 1, b_none + 1.0 / S) - base;
          const int avail = nb == 0 ? S - ks : S;
          fit = (int)std::floor((target - load - base) / per);
          if (fit > avail - 2) fit = avail - 2;
          if (fit < 2) fit = 0;
        }
        if (nb == 0 && fit == 0) {
          if (load > 0.0) { close_cta(); continue; }
          nb = 1;                                       // a target below one block: take it (or what is left of it) whole
        }
        const int e0 = S - ks;                          // block i is still to be swept over K-steps [0, e0)
        if (nb == 0) {                                  // K-steps [e0 - fit, e0) of block i: a middle part
          if (commit) emit_run(st, i, 1, e0, e0 - fit);
          load += cost(st, i, ks, 1, (double)(ks + fit) / S);
          took(st, 1);
          ks += fit;
        } else {
          const int64_t n_run = nb + (fit > 0 ? 1 : 0);
          if (commit) emit_run(st, i, n_run, e0, fit > 0 ? S - fit : 0);
          load += cost(st, i, ks, n_run, fit > 0 ? (double)fit / S : 1.0);
          took(st, n_run);
          i += nb;
          ks = fit;
        }
        close_cta();
      }
    }
    if (commit) for (int k2 = c + 1; k2 <= n_ctas; ++k2) cta_first[k2] = (int)tiles.size();
    return load;
  };
  {
    // feasible = the last CTA does not overshoot.  Feasibility is not quite monotonic in the target (tiles come and go), so after
    // the bisection a scan upwards from a little below looks for a smaller feasible target.
    double lo = 0.5 * total / n_ctas, hi = 2.0 * total / n_ctas + 4096.0;   // assign(hi) never overshoots hi by more than a tile
    for (int it = 0; it < 40; ++it) {
      const double mid = 0.5 * (lo + hi);
      if (assign(mid, false) <= mid + 1e-9) hi = mid; else lo = mid;
    }
    const double from = 0.97 * hi;
    for (int k = 0; k < 120; ++k) {
      const double t = from * (1.0 + 0.00025 * k);
      if (t >= hi) break;
      if (assign(t, false) <= t + 1e-9) { hi = t; break; }
    }
    assign(hi, true);
  }
  const int n_tiles = (int)tiles.size();
  // the epilogue of a CTA's last tile, which nothing hides, is shared with the statistics warps (the HELP instantiation of the kernel;
  // the launch turns it off for the NEXT-2 rider, whose column sums go through one staging buffer)
  sc.help = 1;
  {   // NEXT-2 partial slots: one per block, contiguous per segment (tiles are in row order of their segment already)
    int part = 0;
    for (TcTile& t : tiles) { const int dumped = t.k1 < S * sc.kw ? 1 : 0; t.part0 = part - dumped; part += t.n_blocks - dumped; }   // (a dumped block 0 writes no results)
    sc.n_parts = part;
  }
  TcTile* ht = reinterpret_cast<TcTile*>(h_dst);
  int32_t* hoff = reinterpret_cast<int32_t*>(h_dst + (size_t)n_tiles * sizeof(TcTile));
  for (int i = 0; i < n_tiles; ++i) ht[i] = tiles[i];
  for (int c = 0; c <= n_ctas; ++c) hoff[c] = cta_first[c];
  sc.n_ctas = n_ctas;
  sc.n_tiles = n_tiles;
  sc.d_tiles = reinterpret_cast<const TcTile*>(d_dst);
  sc.d_cta_off = reinterpret_cast<const int32_t*>(d_dst + (size_t)n_tiles * sizeof(TcTile));
  sc.enabled = true;
}

inline cudaError_t tc_set_kernel_attrs() {
  void (*const ks[4])(const TcMaps, const TcParams) = {k_score_tc<1, false>, k_score_tc<2, false>, k_score_tc<1, true>, k_score_tc<2, true>};
  for (auto k : ks) {
    const cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, kTcSmemBytes);
    if (e != cudaSuccess) return e;
  }
  return cudaSuccess;
}

typedef CUresult (*tc_encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                 const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

inline tc_encode_fn tc_get_encode() {
  static tc_encode_fn fn = [] {
    void* f = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &qres) != cudaSuccess || qres != cudaDriverEntryPointSuccess)
      f = nullptr;
    return reinterpret_cast<tc_encode_fn>(f);
  }();
  return fn;
}

// bf16 tensor map over a row-major [rows, d] matrix seen as [d / 64 slices][rows][64 columns] (slice stride 128 B, row stride
// 2 d B): box = [box_slices][box_rows][64 columns], 128-byte swizzle, zero OOB fill.  In shared memory a box is box_slices
// consecutive K-major tiles of box_rows x 128 B, which is what the UMMA descriptors and the statistics warps address.
inline bool tc_make_map(CUtensorMap* m, const void* base, int64_t rows, int d, int box_rows, int box_slices) {
  tc_encode_fn enc = tc_get_encode();
  if (!enc) return false;
  cuuint64_t gdim[3] = {64u, (cuuint64_t)rows, (cuuint64_t)(d / 64)};
  cuuint64_t gstr[2] = {(cuuint64_t)d * 2, 128u};
  cuuint32_t box[3] = {64u, (cuuint32_t)box_rows, (cuuint32_t)box_slices};
  cuuint32_t estr[3] = {1u, 1u, 1u};
  return enc(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(base), gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
             CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// The 20 tensor maps of a launch depend on the (X, Q, R) base pointers only: the plan keeps the last few sets it encoded.
struct TcMapCache {
  struct Entry { const void* X = nullptr; const void* Q = nullptr; const void* R = nullptr; int kw = 0; TcMaps maps; };
  Entry e[4];
  int next = 0;
  const TcMaps* get(const void* X, int64_t N, const void* Q, int64_t nQ, const void* R, int d, int kw) {
    for (Entry& en : e)
      if (en.X == X && en.Q == Q && en.R == R && en.kw == kw) return &en.maps;
    Entry& en = e[next];
    en.X = nullptr;
    for (int k = 0; k < 16; ++k)
      if (!tc_make_map(&en.maps.x[k], X, N, d, 8 * (k + 1), kw)) return nullptr;
    for (int k = 0; k < 3; ++k)
      if (!tc_make_map(&en.maps.q[k], Q, nQ, d, 64 >> k, 1)) return nullptr;
    if (R != nullptr) { if (!tc_make_map(&en.maps.r, R, 64, d, 64, 1)) return nullptr; } else en.maps.r = en.maps.q[0];
    en.X = X; en.Q = Q; en.R = R; en.kw = kw;
    next = (next + 1) & 3;
    return &en.maps;
  }
};

struct TcHeads { float* part; float* m; float bias, tau; };   // NEXT-2 riding the score kernel (Rm = the weight rows W[64, d])

// returns cudaSuccess, or the launch's own error (cudaErrorCooperativeLaunchTooLarge / cudaErrorNotSupported: the cooperative
// launch is not possible on this device / partition and nothing was enqueued), or cudaErrorUnknown if a tensor map could
// not be encoded.
// `q_ready`: two zero-initialised 64-bit words owned by the plan (the kernel leaves them zero).
// `Rm` / `sig` (both NULL = off): NEXT-1, hash rows R[64, d] and the per-token signatures; requires every L <= 64.
// `hf` (NULL = off): NEXT-2, Rm = the head weight rows; same requirement; sig is ignored then.
inline cudaError_t tc_launch_score(const TcSchedule& sc, TcMapCache& cache, const void* X, const void* Q, float* qinv, float* s, float* dnorm,
                                   float* rel, unsigned long long* q_ready, float* xchg, unsigned int* xflag, int64_t N, int64_t nQ, int d, bool inline_qprep, const void* Rm,
                                   unsigned long long* sig, const TcHeads* hf, cudaStream_t st, bool pdl_in = false) {
  const bool rider = sig != nullptr || hf != nullptr;
  const TcMaps* maps = cache.get(X, N, Q, nQ, rider ? Rm : nullptr, d, sc.kw);
  if (!maps) return cudaErrorUnknown;
  TcParams p;
  p.tiles = sc.d_tiles; p.cta_off = sc.d_cta_off; p.qinv = qinv; p.Q = Q; p.nQ = nQ; p.q_ready = q_ready; p.sig = sig; p.s = s; p.dnorm = dnorm; p.rel = rel;
  p.d = d; p.n_kchunks = d / 64; p.kw = sc.kw; p.nx = sc.nx; p.nq = sc.nq; p.qslot_bytes = sc.qslot_bytes; p.wslot = sc.wslot; p.ns = sc.ns;
  p.xchg = xchg; p.xflag = xflag; p.xchg_cols = sc.xchg_cols;
  p.heads_part = hf ? hf->part : nullptr; p.heads_m = hf ? hf->m : nullptr; p.heads_bias = hf ? hf->bias : 0.f; p.heads_tau = hf ? hf->tau : 0.f;
  if (hf) p.sig = nullptr;
  // (no helpers with the NEXT-2 rider: its column sums go through one staging buffer)
  const bool help = sc.help != 0 && hf == nullptr;
  void (*const kern)(const TcMaps, const TcParams) = sc.kw == 2 ? (help ? k_score_tc<2, true> : k_score_tc<2, false>) : (help ? k_score_tc<1, true> : k_score_tc<1, false>);
  if (!inline_qprep) {   // qinv is already there: no CTA waits on another one, a plain launch will do
    p.Q = nullptr;
    return launch_k(kern, dim3((unsigned)sc.n_ctas), dim3(kTcThreads), (size_t)sc.smem_bytes, st, pdl_in, *maps, p);
  }
  // cooperative launch: the query-norm prologue makes the CTAs wait on one another once, so all must be resident
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)sc.n_ctas); cfg.blockDim = dim3(kTcThreads); cfg.dynamicSmemBytes = (size_t)sc.smem_bytes; cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeCooperative;
  attr[0].val.cooperative = 1;
  cfg.attrs = attr; cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kern, *maps, p);
}

}  // namespace msas
