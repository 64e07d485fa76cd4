// k_score_tc.cuh — the Blackwell fast path of the score pass (SURVEY.md §8(a) rows a1+a2+a3 in ONE sweep over X),
// bf16 inputs with d % 64 == 0.
//
//   TMA (cp.async.bulk.tensor, SWIZZLE_128B) stages, per 64-column K-chunk, the token tile X[rows, kc], the matching
//   previous-frame tile X[rows - P, kc] (temporal segments only; an L2 hit, never a second HBM read) and the request's
//   query chunk Q[L, kc] into a multi-stage shared-memory ring.
//   One elected thread issues tcgen05.mma (kind::f16, bf16 x bf16 -> fp32, M = 128, N = pad16(L), K = 16) accumulating
//   S = X·Q^T in TMEM (two accumulators: the epilogue of tile i overlaps the MMAs of tile i+1).          (Eq. 6)
//   Eight CUDA-core warps (two threads per token row and K-slice, half a 128-byte row each: the shorter the time a
//   chunk spends being read, the more of the ring is in flight) read the same shared-memory tiles — conflict-free
//   thanks to the hardware swizzle — and accumulate sum x^2 and sum (x - x_prev)^2 with packed fp32x2 FMAs. (Eq. 3, 5)
//   Four epilogue warps read the accumulator rows with tcgen05.ld (one token row per thread, so the max over query
//   tokens needs no shuffles), scale by 1/|q_j| and 1/|x_i| and write s, sqrt(D), rel: 12 B per token.
//   The temporal ratio gamma = sqrt(D) / (|x_t| + |x_{t-1}|) is finished by the segment kernel, which has both norms
//   from s; the previous row's norm is therefore never recomputed here.
//   The query norms (row a0) are computed by the epilogue warps while the first tile streams in; a non-temporal tile may
//   be a 256-row "double" tile whose two 128-row MMA halves share one query chunk.
//   NEXT-1 (literal LSH probe of Eq. 5): when TcParams::sig is set, 64 hash rows follow the query rows in the B tile and
//   the epilogue packs the signs of their 64 accumulator columns into a per-token signature.
//
// Persistent: one CTA per SM walks a host-built, cost-balanced tile list (round-robin bulk + gap filling).  Tiles never
// straddle a segment.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <queue>
#include <vector>

#include "../../include/msas.h"
#include "msas_internal.cuh"

namespace msas {

struct TcTile {            // 32 bytes
  int32_t row_start;       // global row id of the first row
  int32_t n_rows;          // valid rows, 1..128; up to 256 for a non-temporal "double" tile (two 128-row MMA halves sharing the query
                           // chunk), up to 384 for a "tall" one (three halves; requires pad16(L) <= 64)
  int32_t q_row0;          // first query row of the request
  int32_t L;               // query tokens of the request
  int32_t prev_delta;      // P if the segment is temporal (T > 1), else 0
  int32_t key_rows;        // leading rows of the tile that belong to frame 0 (no previous frame)
  int32_t rank;            // position of the tile when all tiles are sorted by row_start (slot of its learned-head partials)
  int32_t pad_;
};

constexpr int kTcAluSets = 2;                        // ALU warp sets: each takes 8 / kTcAluSets of a row's eight 16-byte units
constexpr int kTcAluUnits = 8 / kTcAluSets;
constexpr int kTcAluWarps = 4 * kTcAluSets;          // per set: one (token row, K-slice) per thread
constexpr int kTcThreads = 256 + 32 * kTcAluWarps;   // 16 warps: 3 single-thread roles, 1 TMEM allocator, 4 epilogue, 8 statistics (roles by scheduler partition: see the kernel)
constexpr int kTcSlots = 16;                         // mbarrier pairs of the chunk ring (slots are variable-sized)
constexpr int kTcBoxBytes = 128 * 128;               // 128 rows x 64 bf16 columns
constexpr int kTcCtrlBytes = 8192;
constexpr int kTcRingBytes = (227 * 1024 - kTcCtrlBytes - 1024 - kTcBoxBytes) & ~1023;   // 1 KB alignment slack, 16 KB MMA over-read pad

struct TcMaps {
  CUtensorMap x[16];   // token rows: box = (16 * (i + 1)) rows x 64 columns, up to the TMA limit of 256 rows
  CUtensorMap q[3];    // query rows: box = 64 / 32 / 16 rows x 64 columns
  CUtensorMap r;       // NEXT-1: the 64 hash rows R[64, d] (box = 64 rows x 64 columns); valid only when TcParams::sig is set
};

struct TcSchedule {
  bool enabled = false;
  bool roles_split = false;      // long temporal sweep: keep the statistics warps off the producers' scheduler partition
  int n_ctas = 0, n_tiles = 0, smem_bytes = 0;
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
  // heads_m[row] = sigmoid(w_0 . x + heads_bias); heads_part[(2 * rank + half) * 64 + c] = per 128-row half of the tile, the
  // number of rows with heads_m < heads_tau (c = 0) and the column sums of w_c . x (c = 1..63); rank = TcTile::rank
  float* heads_part;
  float* heads_m;
  float heads_bias, heads_tau;
  float* s;
  float* dnorm;       // sqrt(sum (x - x_prev)^2) for rows that have a previous frame
  float* rel;
  int d;
  int n_kchunks;
  int roles_split;    // warp-role layout (see the kernel): 1 = the single-thread roles alone on scheduler partition 0
#ifdef MSAS_ABLATE
  int dbg;            // development only: bit0 no ALU math, bit1 no MMA, bit2 no Q loads, bit3 no prev loads
  unsigned long long* dbg_t;
#endif
};

// The chunk ring.  One chunk = one 64-column K-slice of a tile: [x rows16 x 128 B][previous-frame rows, same size,
// temporal tiles only][query rows pad16(L) x 128 B].  Chunks are packed back to back in a circular byte buffer, so a
// short tile (few rows) still leaves the same number of BYTES in flight; every role replays the same deterministic
// offset sequence from the tile list, only the producer tracks which bytes are still in use.
struct TcRing {
  uint32_t off = 0;     // physical byte offset of the next chunk
  uint32_t vhead = 0;   // virtual offset of the next chunk (monotonic mod 2^32, counts wrap padding): only differences are used
  uint32_t k = 0;       // chunk counter -> barrier slot k % kTcSlots, parity (k / kTcSlots) & 1
  __device__ __forceinline__ uint32_t place(uint32_t need) {   // physical offset of the next chunk; advances the ring
    if (off + need > (uint32_t)kTcRingBytes) { vhead += (uint32_t)kTcRingBytes - off; off = 0; }
    const uint32_t r = off;
    off += need; vhead += need;
    return r;
  }
  __device__ __forceinline__ uint32_t slot() const { return k % (uint32_t)kTcSlots; }
  __device__ __forceinline__ uint32_t parity() const { return (k / (uint32_t)kTcSlots) & 1u; }
};
// Geometry of one tile's chunks.  A chunk carries kw consecutive 64-column K-slices so that it holds about 16 KB of
// token rows whatever the tile height (128 rows x 1 slice ... 16 rows x 8 slices): per-chunk costs (barrier round
// trip, producer instructions) are then paid per byte, not per row.  Layout of a chunk:
//   [kw x token slice (xbytes each)] [kw x previous-frame slice, temporal tiles only] [kw x query slice (qbytes each)]
struct TcGeom {
  uint32_t xbytes, xall, qbytes, need;
  int kw, nch, nqb, nqu, nh, hstride;   // nqb = 16-row boxes of B rows (queries + hash rows), nqu = those of the queries alone;
                               // nh = 128-row MMA halves of the tile (2 for a double tile)
  bool has_prev;
};
__device__ __forceinline__ TcGeom tc_geom(const TcTile& t, int nk, int dbg, bool lsh = false) {
  TcGeom g;
  const int rows16 = (t.n_rows + 15) & ~15;
  g.xbytes = (uint32_t)rows16 * 128u;
  g.has_prev = t.prev_delta > 0 && t.key_rows < t.n_rows && !(dbg & 8);
  g.nqu = (dbg & 4) ? 0 : (t.L + 15) >> 4;
  g.nqb = g.nqu + (lsh ? 4 : 0);
  int kw = rows16 <= 16 ? 8 : rows16 <= 32 ? 4 : rows16 <= 64 ? 2 : 1;
  while (kw > 1 && (kw * g.nqb > 16 || nk % kw != 0)) kw >>= 1;   // <= 32 KB of query rows per chunk; kw divides d / 64
  g.kw = kw;
  g.nh = (rows16 + 127) >> 7;            // 3 = a TALL tile (257..384 rows): only where pad16(L) <= 64, accumulator halves 64 columns apart
  g.hstride = g.nh > 2 ? 64 : 128;
  g.nch = nk / kw;
  g.xall = g.xbytes * (g.has_prev ? 2u : 1u);
  g.qbytes = (uint32_t)g.nqb * 2048u;
  g.need = (uint32_t)kw * (g.xall + g.qbytes);
  return g;
}

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
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* map, uint32_t bar, int c0, int c1) {
  asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];" ::"r"(dst),
               "l"(map), "r"(bar), "r"(c0), "r"(c1)
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
  uint64_t full[kTcSlots];           // TMA -> consumers           (1 arrival + transaction bytes)
  uint64_t empty[kTcSlots];          // consumers -> TMA           (1 MMA commit + the ALU warps)
  uint64_t tmem_full[2];             // MMA -> epilogue            (1 commit)
  uint64_t tmem_empty[2];            // epilogue -> MMA            (4 warps)
  uint64_t stat_full[2];             // ALU -> epilogue            (ALU warps)
  uint64_t stat_empty[2];            // epilogue -> ALU            (4 warps)
  uint32_t tmem_base;
  uint32_t pad_[31];
  float rowstat[2][kTcAluSets][2][128];   // partial sum x^2, sum (x - x_prev)^2 per (ALU set, K-slice, tile row), double buffered
  union {
    float hred[2][4][64];            // NEXT-2: per-warp column sums of the 64 head columns, double buffered (never on tall tiles)
    float rowstat3[2][kTcAluSets][128];   // tall tiles: partial sum x^2 of the third half's rows (half a row per ALU set), double buffered
  };
};
static_assert(sizeof(TcCtrl) <= kTcCtrlBytes, "control block too large");

__global__ void __launch_bounds__(kTcThreads, 1)
k_score_tc(const __grid_constant__ TcMaps maps, const TcParams p) {
  const CUtensorMap& mx128 = maps.x[7];
  const CUtensorMap& mq64 = maps.q[0];
  const CUtensorMap& mq32 = maps.q[1];
  const CUtensorMap& mq16 = maps.q[2];
  extern __shared__ unsigned char smem_raw[];
  unsigned char* smem = reinterpret_cast<unsigned char*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  TcCtrl* ctrl = reinterpret_cast<TcCtrl*>(smem);
  unsigned char* ring0 = smem + kTcCtrlBytes;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  // Warp roles by scheduler partition (SMSP = warp % 4).  The three single-thread roles that keep the pipeline fed share SMSP 0
  // with one (mostly waiting) epilogue warp, so the arithmetic warps never compete with them for issue slots:
  //   SMSP 0: warp 0 TMA token rows, warp 4 TMA query rows, warp 8 MMA issuer, warp 12 epilogue (TMEM lanes 0-31)
  //   SMSP 1-3: warps 1, 2, 3 epilogue (lane quarter = warp % 4); warps 5-7, 9-11, 13, 14 statistics; warp 15 TMEM allocation
  // That helps long temporal sweeps (config 3: -5 %), where the statistics warps are busiest; elsewhere two statistics warps
  // per partition (roles_split = 0: warps 0 TMA X, 1 MMA, 2 TMEM, 3 TMA Q, 4-7 epilogue, 8-15 statistics) measure 2 % faster.
  const bool split = p.roles_split != 0;
  const bool is_xprod = warp == 0, is_qprod = warp == (split ? 4 : 3), is_mma = warp == (split ? 8 : 1), is_tmem = warp == (split ? 15 : 2);
  const bool is_epi = split ? (warp == 12 || (warp >= 1 && warp <= 3)) : (warp >= 4 && warp < 8);
  const bool is_alu = !is_xprod && !is_qprod && !is_mma && !is_tmem && !is_epi;
  const int alu_idx = !split ? warp - 8 : warp < 8 ? warp - 5 : warp < 12 ? warp - 6 : warp - 7;   // split: 5,6,7 -> 0..2; 9,10,11 -> 3..5; 13,14 -> 6,7
  const int tile_lo = p.cta_off[blockIdx.x], tile_hi = p.cta_off[blockIdx.x + 1];
  const int nk = p.n_kchunks;
  const bool lsh = p.sig != nullptr || p.heads_part != nullptr;   // 64 more B rows after the query rows (hash rows or head weights)
#ifdef MSAS_ABLATE
  const int dbg = p.dbg;
  auto gtime = [] { unsigned long long t; asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t)); return t; };
  if (tid == 0 && p.dbg_t) { p.dbg_t[blockIdx.x * 8 + 0] = gtime(); unsigned sm; asm volatile("mov.u32 %0, %smid;" : "=r"(sm)); p.dbg_t[blockIdx.x * 8 + 1] = sm; }
#else
  constexpr int dbg = 0;
#endif

  pdl_launch_dependents();   // the segment kernel may be scheduled as SMs free up; it waits for this grid to complete
  if (is_mma && lane == 0) {
    for (int i = 0; i < kTcSlots; ++i) { mbar_init(smem_u32(&ctrl->full[i]), 2); mbar_init(smem_u32(&ctrl->empty[i]), 1 + kTcAluWarps); }
    for (int i = 0; i < 2; ++i) {
      mbar_init(smem_u32(&ctrl->tmem_full[i]), 1); mbar_init(smem_u32(&ctrl->tmem_empty[i]), 4);
      mbar_init(smem_u32(&ctrl->stat_full[i]), kTcAluWarps); mbar_init(smem_u32(&ctrl->stat_empty[i]), 4);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (is_tmem) {   // TMEM: 2 tiles in flight x 2 halves x 128 fp32 columns (all 512 columns: one CTA per SM)
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&ctrl->tmem_base)), "r"(512) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  if (is_xprod && lane == 0) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(&mx128) : "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(&mq64) : "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(&mq16) : "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = ctrl->tmem_base;
  pdl_wait();   // plain (non-cooperative) launches are chained behind k_qprep: the set-up above overlaps its tail

  if (is_xprod || is_qprod) {
    // ===================================================================== TMA producers (one thread each)
    // warp 0 streams the token rows (and the previous-frame rows), warp 3 the query rows.  A single thread issues about
    // one instruction every few cycles, so the per-chunk loop is kept to a few dozen instructions per producer.
    if (lane == 0) {
      const bool xprod = is_xprod;
      TcRing ring;
      // `tail` replays the same placement sequence one released chunk at a time: tail.vhead is (a lower bound of) the
      // virtual start of the oldest chunk whose release has not been observed yet, tail.k its index.  Registers only.
      TcRing tail;
      int tail_t = tile_lo, tail_ch = 0;
      TcGeom tg = tc_geom(p.tiles[tile_lo], nk, dbg, lsh);
      for (int t = tile_lo; t < tile_hi; ++t) {
        const TcTile tile = p.tiles[t];
        const TcGeom g = tc_geom(tile, nk, dbg, lsh);
        const bool tall = g.nh > 2;                                 // 257..384 rows: a 256-row box and a second one for the rest
        const CUtensorMap* mx = &maps.x[((tall ? 32768u : g.xbytes) >> 11) - 1];      // one box of rows16 rows per K-slice
        const CUtensorMap* mx2 = &maps.x[tall ? ((g.xbytes - 32768u) >> 11) - 1 : 0];
        const int row = tile.row_start, prow = tile.row_start - tile.prev_delta;
        const uint32_t poff = (uint32_t)g.kw * g.xbytes;            // previous-frame slices follow the token slices
#ifdef MSAS_ABLATE
        if (xprod && (blockIdx.x == 0 || blockIdx.x == 77) && p.dbg_t) p.dbg_t[2048 + (blockIdx.x ? 64 : 0) + (t - tile_lo)] = gtime();
#endif
        for (int ch = 0; ch < g.nch; ++ch) {
          const uint32_t off = ring.place(g.need);
          // wait until the barrier slot is free and the bytes of this chunk no longer overlap an unreleased chunk
          while (tail.k < ring.k && (ring.k - tail.k >= (uint32_t)kTcSlots || ring.vhead - tail.vhead > (uint32_t)kTcRingBytes)) {
            mbar_wait(smem_u32(&ctrl->empty[tail.slot()]), tail.parity());
            tail.place(tg.need);
            ++tail.k;
            if (++tail_ch == tg.nch && tail_t + 1 < tile_hi) { tail_ch = 0; tg = tc_geom(p.tiles[++tail_t], nk, dbg, lsh); }
          }
          const uint32_t bar = smem_u32(&ctrl->full[ring.slot()]);
          const uint32_t base = smem_u32(ring0 + off);
          if (xprod) {
            const bool ld_prev = g.has_prev;
            mbar_expect_tx(bar, (uint32_t)g.kw * (ld_prev ? g.xall : g.xbytes));
            for (int j = 0; j < g.kw; ++j) {
              const int c0 = (ch * g.kw + j) * 64;
              const uint32_t dst = base + (uint32_t)j * g.xbytes;
              tma_load_2d(dst, mx, bar, c0, row);      // rows past the end of X are zero-filled by the TMA unit
              if (tall) tma_load_2d(dst + 32768u, mx2, bar, c0, row + 256);
              if (ld_prev) tma_load_2d(dst + poff, mx, bar, c0, prow);
            }
          } else {
            mbar_expect_tx(bar, (uint32_t)g.kw * g.qbytes);
            uint32_t sq = base + (uint32_t)g.kw * g.xall;
            for (int j = 0; j < g.kw; ++j) {
              const int c0 = (ch * g.kw + j) * 64;
              int qr = tile.q_row0;
              for (int i = 0; i < (g.nqu >> 2); ++i) { tma_load_2d(sq, &mq64, bar, c0, qr); sq += 8192; qr += 64; }
              if (g.nqu & 2) { tma_load_2d(sq, &mq32, bar, c0, qr); sq += 4096; qr += 32; }
              if (g.nqu & 1) { tma_load_2d(sq, &mq16, bar, c0, qr); sq += 2048; }
              if (lsh) { tma_load_2d(sq, &maps.r, bar, c0, 0); sq += 8192; }   // the hash rows follow the query rows: one B tile
            }
          }
          ++ring.k;
        }
      }
    }
  } else if (is_mma) {
    // ===================================================================== MMA issuer (one thread)
    if (lane == 0) {
      TcRing ring;
      int it = 0;
      for (int t = tile_lo; t < tile_hi; ++t, ++it) {
        const TcTile tile = p.tiles[t];
        const TcGeom g = tc_geom(tile, nk, dbg, lsh);
        const uint32_t idesc = umma_idesc_bf16(g.nqb << 4);   // N = pad16(L) (+ 64 hash rows)
        const int acc = it & 1;
        const uint32_t acc_phase = (uint32_t)(it >> 1) & 1u;
        mbar_wait(smem_u32(&ctrl->tmem_empty[acc]), acc_phase ^ 1u);
        tc_fence_after();
        const uint32_t d_tmem = tmem_base + (uint32_t)acc * 256u;
        for (int ch = 0; ch < g.nch; ++ch) {
          const uint32_t off = ring.place(g.need);
          mbar_wait(smem_u32(&ctrl->full[ring.slot()]), ring.parity());
          tc_fence_after();
          const uint32_t base = smem_u32(ring0 + off);
          if (!(dbg & 2)) {
            for (int j = 0; j < g.kw; ++j) {
              const uint64_t bdesc = umma_desc_sw128(base + (uint32_t)g.kw * g.xall + (uint32_t)j * g.qbytes);
              for (int h = 0; h < g.nh; ++h) {
                // M = 128: rows past the tile read whatever follows in the ring (their accumulator rows are never used)
                const uint64_t adesc = umma_desc_sw128(base + (uint32_t)j * g.xbytes + (uint32_t)h * (uint32_t)kTcBoxBytes);
#pragma unroll
                for (int k = 0; k < 4; ++k)   // 4 x K=16 inside the 128-byte swizzle atom: +32 B = +2 in the 16-byte address field
                  tc_mma_bf16(d_tmem + (uint32_t)(h * g.hstride), adesc + (uint64_t)(2 * k), bdesc + (uint64_t)(2 * k), idesc, (uint32_t)(ch | j | k));
              }
            }
          }
          tc_commit(smem_u32(&ctrl->empty[ring.slot()]));
          ++ring.k;
        }
        tc_commit(smem_u32(&ctrl->tmem_full[acc]));
      }
    }
  } else if (is_epi) {
    // ===================================================================== epilogue: one accumulator row per thread
    const int q = warp & 3;                  // TMEM lane quarter this warp may access (warp % 4)
    const int r = q * 32 + lane;             // tile row
    const float inv_d = 1.0f / (float)p.d;
    // a0 inside the same launch: while the first tile streams in, these four warps compute 1 / |q_j| for this CTA's
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
    bool q_ok = p.Q == nullptr;
    int it = 0;
    for (int t = tile_lo; t < tile_hi; ++t, ++it) {
      const TcTile tile = p.tiles[t];
      const TcGeom g = tc_geom(tile, nk, dbg, lsh);
      const int acc = it & 1;
      const uint32_t ph = (uint32_t)(it >> 1) & 1u;
      const int nqb = (tile.L + 15) >> 4;
      const float* qinv = p.qinv + tile.q_row0;
      mbar_wait(smem_u32(&ctrl->tmem_full[acc]), ph);
      tc_fence_after();
      if (!q_ok) {   // all CTAs' shares of qinv are written (first tile only; normally long since true)
        unsigned long long seen;
        do { asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(seen) : "l"(p.q_ready) : "memory"); } while (seen < (unsigned long long)gridDim.x);
        q_ok = true;
      }
      float m[3] = {-INFINITY, -INFINITY, -INFINITY};   // per 128-row half of the tile
#pragma unroll
      for (int h = 0; h < 3; ++h)
        for (int cb = 0; cb < (h < g.nh ? nqb : 0); ++cb) {
          uint32_t v[16];
          tc_ld16(tmem_base + (uint32_t)acc * 256u + (uint32_t)(h * g.hstride) + (uint32_t)cb * 16u + ((uint32_t)(q * 32) << 16), v);
          tc_wait_ld();
#pragma unroll
          for (int j = 0; j < 16; ++j) {
            const int col = cb * 16 + j;
            if (col < tile.L) m[h] = fmaxf(m[h], __uint_as_float(v[j]) * qinv[col]);
          }
        }
      if (p.heads_part != nullptr) {   // NEXT-2: column 0 -> the learned spatial map, all 64 -> per-half column sums (fixed order)
#pragma unroll 1
        for (int h = 0; h < 2; ++h) {
          float tot[2] = {0.f, 0.f};
          if (h < g.nh) {
            const int tr = h * 128 + r;
            const bool valid = tr < tile.n_rows;
#pragma unroll
            for (int grp = 0; grp < 2; ++grp) {
              float x[32];
#pragma unroll
              for (int cb = 0; cb < 2; ++cb) {
                uint32_t v[16];
                tc_ld16(tmem_base + (uint32_t)acc * 256u + (uint32_t)h * 128u + (uint32_t)(g.nqu + grp * 2 + cb) * 16u + ((uint32_t)(q * 32) << 16), v);
                tc_wait_ld();
#pragma unroll
                for (int j = 0; j < 16; ++j) x[cb * 16 + j] = valid ? __uint_as_float(v[j]) : 0.f;
              }
              if (grp == 0) {
                float below = 0.f;
                if (valid) {
                  const float M = sigmoidf_acc(x[0] + p.heads_bias);
                  p.heads_m[(int64_t)tile.row_start + tr] = M;
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
          }
          const int hb = (it * 2 + h) & 1;
          ctrl->hred[hb][q][lane] = tot[0];
          ctrl->hred[hb][q][32 + lane] = tot[1];
          asm volatile("bar.sync 1, 128;" ::: "memory");       // the four epilogue warps
          if (r < 64)
            p.heads_part[((int64_t)tile.rank * 2 + h) * 64 + r] = (ctrl->hred[hb][0][r] + ctrl->hred[hb][1][r]) + (ctrl->hred[hb][2][r] + ctrl->hred[hb][3][r]);
        }
      } else if (lsh) {   // NEXT-1: the 64 accumulator columns after the query columns are r_k . x: their signs are the hash bits
        for (int h = 0; h < g.nh; ++h) {
          unsigned long long bits = 0ull;
#pragma unroll
          for (int cb = 0; cb < 4; ++cb) {
            uint32_t v[16];
            tc_ld16(tmem_base + (uint32_t)acc * 256u + (uint32_t)h * 128u + (uint32_t)(g.nqu + cb) * 16u + ((uint32_t)(q * 32) << 16), v);
            tc_wait_ld();
#pragma unroll
            for (int j = 0; j < 16; ++j) bits |= (unsigned long long)(__uint_as_float(v[j]) >= 0.f) << (cb * 16 + j);
          }
          const int tr = h * 128 + r;
          if (tr < tile.n_rows) p.sig[(int64_t)tile.row_start + tr] = bits;
        }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(smem_u32(&ctrl->tmem_empty[acc]));
      mbar_wait(smem_u32(&ctrl->stat_full[acc]), ph);
      float n2[3] = {0.f, 0.f, 0.f}, D[3] = {0.f, 0.f, 0.f};
      if (g.nh >= 2) {                       // double tile: ALU thread `row` holds the whole row's sums, row = set * 128 + r
#pragma unroll
        for (int h = 0; h < 2; ++h) { n2[h] = ctrl->rowstat[acc][h][0][r]; D[h] = ctrl->rowstat[acc][h][1][r]; }
        if (g.nh > 2) n2[2] = ctrl->rowstat3[acc][0][r] + ctrl->rowstat3[acc][1][r];   // third half: half a row per ALU set
      } else if (r < tile.n_rows) {          // one partial per (ALU set, K-slice of the chunk, row)
        const int rp2 = 128 / g.kw;
        for (int j = 0; j < g.kw; ++j)
#pragma unroll
          for (int st = 0; st < kTcAluSets; ++st) { n2[0] += ctrl->rowstat[acc][st][0][r + j * rp2]; D[0] += ctrl->rowstat[acc][st][1][r + j * rp2]; }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(smem_u32(&ctrl->stat_empty[acc]));
#pragma unroll
      for (int h = 0; h < 3; ++h) {
        const int tr = h * 128 + r;
        if (h < g.nh && tr < tile.n_rows) {
          const int64_t row = (int64_t)tile.row_start + tr;
          p.s[row] = sqrtf(n2[h] * inv_d);
          p.dnorm[row] = sqrtf(D[h]);
          p.rel[row] = n2[h] > 0.f ? m[h] / sqrtf(n2[h]) : 0.f;
        }
      }
    }
  } else if (is_alu) {
    // ===================================================================== CUDA-core statistics: one thread per (row, K-slice)
    const int a = (alu_idx & 3) * 32 + lane;
    const uint32_t set = (uint32_t)alu_idx >> 2;          // which share of the row's eight 16-byte units this thread reads
    TcRing ring;
    int it = 0;
    for (int t = tile_lo; t < tile_hi; ++t, ++it) {
      const TcTile tile = p.tiles[t];
      const TcGeom g = tc_geom(tile, nk, dbg, lsh);
      const int rp2 = 128 / g.kw;
      const bool dbl = g.nh >= 2;                        // double tile: 256 threads = 256 rows, a whole row each, no previous frame
      const bool act3 = g.nh > 2 && 256 + a < tile.n_rows && !(dbg & 1);   // tall tile: row 256 + a, half of it per ALU set
      uint64_t n3a = 0, n3b = 0;
      const int r = dbl ? (int)set * 128 + a : (a & (rp2 - 1)), j = dbl ? 0 : a / rp2;
      const bool active = r < tile.n_rows && !(dbg & 1);
      // hardware 128-byte swizzle: 16-byte unit u of row r sits at unit u ^ (r & 7)
      const uint32_t my_off = (uint32_t)j * g.xbytes + (uint32_t)r * 128u;
      const uint32_t sw = (uint32_t)(r & 7);
      const uint32_t poff = (uint32_t)g.kw * g.xbytes;
      uint64_t n2a = 0, n2b = 0, Da = 0, Db = 0;     // packed fp32 pairs, all zero bits = (0.f, 0.f)
      for (int ch = 0; ch < g.nch; ++ch) {
        const uint32_t off = ring.place(g.need);
        mbar_wait(smem_u32(&ctrl->full[ring.slot()]), ring.parity());
#ifdef MSAS_ABLATE
        if (alu_idx == 0 && lane == 0 && p.dbg_t && t == tile_lo && ch == 0) p.dbg_t[blockIdx.x * 8 + 2] = gtime();
#endif
        if (active && dbl) {
          const unsigned char* sx = ring0 + off + my_off;
          uint4 x[8];
#pragma unroll
          for (int u = 0; u < 8; ++u) x[u] = *reinterpret_cast<const uint4*>(sx + (((uint32_t)u ^ sw) << 4));
#pragma unroll
          for (int u = 0; u < 8; ++u) {
            fma_sq_f32x2(n2a, bf16x2_to_f32x2(x[u].x)); fma_sq_f32x2(n2b, bf16x2_to_f32x2(x[u].y));
            fma_sq_f32x2(n2a, bf16x2_to_f32x2(x[u].z)); fma_sq_f32x2(n2b, bf16x2_to_f32x2(x[u].w));
          }
          if (act3) {
            const unsigned char* s3 = ring0 + off + (uint32_t)(256 + a) * 128u;
            const uint32_t u3 = set * (uint32_t)kTcAluUnits, sw3 = (uint32_t)(a & 7);
            uint4 y[kTcAluUnits];
#pragma unroll
            for (int u = 0; u < kTcAluUnits; ++u) y[u] = *reinterpret_cast<const uint4*>(s3 + (((u3 + (uint32_t)u) ^ sw3) << 4));
#pragma unroll
            for (int u = 0; u < kTcAluUnits; ++u) {
              fma_sq_f32x2(n3a, bf16x2_to_f32x2(y[u].x)); fma_sq_f32x2(n3b, bf16x2_to_f32x2(y[u].y));
              fma_sq_f32x2(n3a, bf16x2_to_f32x2(y[u].z)); fma_sq_f32x2(n3b, bf16x2_to_f32x2(y[u].w));
            }
          }
        } else if (active) {
          const unsigned char* sx = ring0 + off + my_off;
          uint4 x[kTcAluUnits];
          const uint32_t u0 = set * (uint32_t)kTcAluUnits;       // this set's share of the row's eight 16-byte units
#pragma unroll
          for (int u = 0; u < kTcAluUnits; ++u) x[u] = *reinterpret_cast<const uint4*>(sx + (((u0 + (uint32_t)u) ^ sw) << 4));
          if (g.has_prev && !(dbg & 16)) {
            const unsigned char* su = sx + poff;
            uint4 v[kTcAluUnits];
#pragma unroll
            for (int u = 0; u < kTcAluUnits; ++u) v[u] = *reinterpret_cast<const uint4*>(su + (((u0 + (uint32_t)u) ^ sw) << 4));
            if (dbg & 32) {   // development only: the loads without the arithmetic
#pragma unroll
              for (int u = 0; u < kTcAluUnits; ++u) n2a ^= (uint64_t)(x[u].x ^ x[u].y ^ x[u].z ^ x[u].w ^ v[u].x ^ v[u].y ^ v[u].z ^ v[u].w);
            } else
#pragma unroll
            for (int u = 0; u < kTcAluUnits; ++u) {
              const uint64_t x0 = bf16x2_to_f32x2(x[u].x), x1 = bf16x2_to_f32x2(x[u].y), x2 = bf16x2_to_f32x2(x[u].z), x3 = bf16x2_to_f32x2(x[u].w);
              const uint64_t e0 = sub_f32x2(x0, bf16x2_to_f32x2(v[u].x)), e1 = sub_f32x2(x1, bf16x2_to_f32x2(v[u].y));
              const uint64_t e2 = sub_f32x2(x2, bf16x2_to_f32x2(v[u].z)), e3 = sub_f32x2(x3, bf16x2_to_f32x2(v[u].w));
              fma_sq_f32x2(n2a, x0); fma_sq_f32x2(n2b, x1); fma_sq_f32x2(n2a, x2); fma_sq_f32x2(n2b, x3);
              fma_sq_f32x2(Da, e0); fma_sq_f32x2(Db, e1); fma_sq_f32x2(Da, e2); fma_sq_f32x2(Db, e3);
            }
          } else {
#pragma unroll
            for (int u = 0; u < kTcAluUnits; ++u) {
              fma_sq_f32x2(n2a, bf16x2_to_f32x2(x[u].x)); fma_sq_f32x2(n2b, bf16x2_to_f32x2(x[u].y));
              fma_sq_f32x2(n2a, bf16x2_to_f32x2(x[u].z)); fma_sq_f32x2(n2b, bf16x2_to_f32x2(x[u].w));
            }
          }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(smem_u32(&ctrl->empty[ring.slot()]));
        ++ring.k;
      }
      const float n2 = sum_f32x2(n2a) + sum_f32x2(n2b);
      const float D = sum_f32x2(Da) + sum_f32x2(Db);
      const int buf = it & 1;
      const uint32_t ph = (uint32_t)(it >> 1) & 1u;
      mbar_wait(smem_u32(&ctrl->stat_empty[buf]), ph ^ 1u);
      ctrl->rowstat[buf][set][0][a] = n2; ctrl->rowstat[buf][set][1][a] = D;      // slot a = j * rp2 + r
      if (g.nh > 2) ctrl->rowstat3[buf][set][a] = sum_f32x2(n3a) + sum_f32x2(n3b);
      __syncwarp();
      if (lane == 0) mbar_arrive(smem_u32(&ctrl->stat_full[buf]));
    }
  }

  tc_fence_before();
  __syncthreads();
#ifdef MSAS_ABLATE
  if (tid == 0 && p.dbg_t) p.dbg_t[blockIdx.x * 8 + 3] = gtime();
#endif
  if (tid == 0 && p.Q != nullptr) {   // every CTA is past its wait on q_ready[0] by now; the last one out zeroes both counters
    __threadfence();
    if (atomicAdd(p.q_ready + 1, 1ull) == (unsigned long long)gridDim.x - 1ull) { p.q_ready[0] = 0ull; p.q_ready[1] = 0ull; __threadfence(); }
  }
  if (is_tmem) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(512) : "memory");
  }
}

// ------------------------------------------------------------------------------------------------ host side
// Schedule.  Cost of a tile = bytes it pulls into the SM in units of 128-byte rows: rows16 from HBM, the previous-frame
// rows and the query rows from L2 at a fraction of that.  Two phases:
//   bulk: 128-row tiles dealt round-robin in row order, as many complete rounds as fit under the per-CTA target
//         (neighbouring CTAs sweep neighbouring rows at the same time, so previous-frame tiles are still in L2);
//   fill: the remaining rows are cut into tiles sized to each CTA's remaining gap (largest gap first, multiples of 16
//         rows, at least 32 unless a segment ends), which levels the CTAs to about one 16-row box.
// Short tiles keep the same bytes in flight (variable-size chunk ring) but re-stream the query chunks more often,
// which is why only the fill phase uses them.
struct TcCost {
  double w_prev = 0.25, w_q = 0.70, c_tile = 50.0;   // fitted to CTA finish times: ~27 us per MB of token rows, 12-19 us per MB of query rows, several us per tile
  int roles = -1;              // development override of the warp-role layout (-1 = by the schedule)
  int hmax_plain = 256, hmax_tall = 384;   // tallest non-temporal tile; tall = three MMA halves, where pad16(L) <= 64
  TcCost() {
#ifdef MSAS_ABLATE
    if (getenv("MSAS_HTALL")) hmax_tall = atoi(getenv("MSAS_HTALL"));
    if (getenv("MSAS_ROLES")) roles = atoi(getenv("MSAS_ROLES"));
    if (getenv("MSAS_HMAX")) hmax_plain = atoi(getenv("MSAS_HMAX"));
    if (getenv("MSAS_WPREV")) w_prev = atof(getenv("MSAS_WPREV"));
    if (getenv("MSAS_WQ")) w_q = atof(getenv("MSAS_WQ"));
    if (getenv("MSAS_CTILE")) c_tile = atof(getenv("MSAS_CTILE"));
#endif
  }
};
inline size_t tc_max_tiles(const mas_segment* segs, int32_t n_segs) {
  size_t tiles = 0;   // upper bound: every segment in 32-row tiles plus one remainder each
  for (int32_t k = 0; k < n_segs; ++k) tiles += (size_t)(((int64_t)segs[k].n_frames * segs[k].n_patches + 31) / 32) + 1;
  return tiles;
}
inline size_t tc_schedule_bytes(const mas_segment* segs, int32_t n_segs) {
  return tc_max_tiles(segs, n_segs) * sizeof(TcTile) + 1024 * sizeof(int32_t) + 256;
}

// Builds the tile list (grouped per CTA) and the per-CTA offsets into `h_dst`; `d_dst` is where the image will live.
inline void tc_build_schedule(TcSchedule& sc, const mas_segment* segs, int32_t n_segs, const int64_t* q_off, int32_t d, int32_t dtype,
                              int sm_count, char* h_dst, char* d_dst, bool tall_tiles = true) {
  sc = TcSchedule();
  if (dtype != MAS_BF16 || d % 64 != 0 || sm_count < 1 || sm_count > 1000) return;
  const TcCost cw;
  struct SegInfo { double w_row, c_fix; int L, P, hmax; };   // hmax: tallest tile (256 = double tile, non-temporal only)
  std::vector<SegInfo> si(n_segs);
  double total = 0.0;
  int64_t n_full = 0;
  for (int32_t k = 0; k < n_segs; ++k) {
    const mas_segment& s = segs[k];
    const int64_t n = (int64_t)s.n_frames * s.n_patches;
    si[k].L = (int)(q_off[s.request + 1] - q_off[s.request]);
    si[k].P = s.n_frames > 1 ? s.n_patches : 0;
    si[k].w_row = 1.0 + (si[k].P > 0 ? cw.w_prev : 0.0);
    // tall tiles (three MMA halves, 48 KB chunks) pay where they save a tile of a SHORT segment (a 576-token image: 2 tiles
    // instead of 3); on long segments the double tile keeps more chunks in flight (measured: ragged mix +2 % with tall tiles)
    si[k].hmax = si[k].P > 0 ? 128 : (tall_tiles && si[k].L <= 64 && n <= 2 * cw.hmax_tall ? std::max(cw.hmax_plain, cw.hmax_tall) : cw.hmax_plain);
    si[k].c_fix = cw.w_q * (((si[k].L + 15) / 16) * 16) + cw.c_tile;
    total += (double)n * si[k].w_row + (double)((n + si[k].hmax - 1) / si[k].hmax) * si[k].c_fix;
    n_full += n / si[k].hmax;
  }
  const int n_ctas = (int)std::min<int64_t>(sm_count, std::max<int64_t>(1, (int64_t)(total / 64.0)));

  std::vector<TcTile> tiles;
  std::vector<std::vector<int>> per;
  auto make_tile = [&](int32_t k, int64_t r, int h) {
    const mas_segment& s = segs[k];
    TcTile t{};
    t.row_start = (int32_t)(s.row0 + r);
    t.n_rows = h;
    t.q_row0 = (int32_t)q_off[s.request];
    t.L = si[k].L;
    t.prev_delta = si[k].P;
    t.key_rows = si[k].P > 0 ? (int32_t)std::min<int64_t>(std::max<int64_t>(si[k].P - r, 0), h) : 0;
    tiles.push_back(t);
    return (int)tiles.size() - 1;
  };
  double cost128_max = 0.0;
  for (int32_t k = 0; k < n_segs; ++k) cost128_max = std::max(cost128_max, (double)si[k].hmax * si[k].w_row + si[k].c_fix);
  struct Piece { int32_t seg; int64_t r0, r1; };
  // one attempt at per-CTA target `target`; returns the heaviest CTA's load
  auto attempt = [&](double target) {
    tiles.clear();
    per.assign(n_ctas, std::vector<int>());
    std::vector<double> load(n_ctas, 0.0);
    // ---- bulk: complete round-robin rounds of 128-row tiles that keep every CTA under target - reserve
    const double reserve = 48.0;
    int64_t rounds = (int64_t)((target - reserve) / cost128_max);
    if (rounds < 0) rounds = 0;
    const int64_t n_bulk = std::min<int64_t>(n_full, rounds * n_ctas) / n_ctas * n_ctas;
    std::vector<Piece> pieces;
    int64_t dealt = 0;
    for (int32_t k = 0; k < n_segs; ++k) {
      const int64_t n = (int64_t)segs[k].n_frames * segs[k].n_patches;
      int64_t r = 0;
      while (n - r >= si[k].hmax && dealt < n_bulk) {
        const int c = (int)(dealt % n_ctas);
        per[c].push_back(make_tile(k, r, si[k].hmax));
        load[c] += (double)si[k].hmax * si[k].w_row + si[k].c_fix;
        r += si[k].hmax; ++dealt;
      }
      if (r < n) pieces.push_back(Piece{k, r, n});
    }
    // ---- fill: cut the remaining rows to the CTAs' gaps, largest gap first
    typedef std::pair<double, int> Gap;   // (gap, -cta) : max-heap, ties -> lowest CTA id
    std::priority_queue<Gap> heap;
    for (int c = 0; c < n_ctas; ++c) heap.push(Gap(target - load[c], -c));
    for (const Piece& pc : pieces) {
      const SegInfo& g = si[pc.seg];
      int64_t r = pc.r0;
      while (r < pc.r1) {
        const Gap top = heap.top(); heap.pop();
        const int c = -top.second;
        const int64_t left = pc.r1 - r;
        int64_t h = (int64_t)((top.first - g.c_fix) / g.w_row) / 16 * 16;
        h = std::max<int64_t>(32, std::min<int64_t>(g.hmax, h));
        if (h >= left || left - h < 32) h = std::min<int64_t>(left, g.hmax);
        per[c].push_back(make_tile(pc.seg, r, (int)h));
        load[c] += (double)((h + 15) / 16 * 16) * g.w_row + g.c_fix;
        heap.push(Gap(target - load[c], -c));
        r += h;
      }
    }
    return *std::max_element(load.begin(), load.end());
  };
  // the fill phase spends a per-tile cost the estimate above cannot know: raise the target until no CTA overshoots
  double best_t = total / n_ctas, best_max = 1e300;
  for (int i = 0; i < 40; ++i) {
    const double t = total / n_ctas * (1.0 + 0.005 * i);
    const double m = attempt(t);
    if (m < best_max - 1e-9) { best_max = m; best_t = t; }
  }
  attempt(best_t);
  const int n_tiles = (int)tiles.size();
  TcTile* ht = reinterpret_cast<TcTile*>(h_dst);
  int32_t* hoff = reinterpret_cast<int32_t*>(h_dst + (size_t)n_tiles * sizeof(TcTile));
  int w = 0;
  for (int c = 0; c < n_ctas; ++c) {
    std::sort(per[c].begin(), per[c].end(), [&](int a, int b) { return tiles[a].row_start < tiles[b].row_start; });
    hoff[c] = w;
    for (int i : per[c]) ht[w++] = tiles[i];
  }
  hoff[n_ctas] = w;
  {   // rank of every tile in row order: tiles never straddle segments, so a segment's tiles are one contiguous rank range
    std::vector<int> order(n_tiles);
    for (int i = 0; i < n_tiles; ++i) order[i] = i;
    std::sort(order.begin(), order.end(), [&](int a, int b) { return ht[a].row_start < ht[b].row_start; });
    for (int i = 0; i < n_tiles; ++i) ht[order[i]].rank = i;
  }
  sc.smem_bytes = kTcCtrlBytes + 1024 + kTcRingBytes + kTcBoxBytes;
  sc.n_ctas = n_ctas;
  sc.n_tiles = n_tiles;
  sc.d_tiles = reinterpret_cast<const TcTile*>(d_dst);
  sc.d_cta_off = reinterpret_cast<const int32_t*>(d_dst + (size_t)n_tiles * sizeof(TcTile));
  {   // warp-role layout: see the kernel
    int64_t rows = 0, rows_prev = 0;
    for (int i = 0; i < n_tiles; ++i) { rows += ht[i].n_rows; if (ht[i].prev_delta > 0 && ht[i].key_rows < ht[i].n_rows) rows_prev += ht[i].n_rows; }
    sc.roles_split = cw.roles >= 0 ? cw.roles != 0 : (rows_prev * 10 >= rows * 4 && n_tiles >= 4 * n_ctas);
  }
  sc.enabled = true;
}

inline void tc_set_kernel_attrs() { cudaFuncSetAttribute(k_score_tc, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024); }

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

// 2-D bf16 tensor map over a row-major [rows, d] matrix, box = [box_rows, 64 columns], 128-byte swizzle, zero OOB fill.
inline bool tc_make_map(CUtensorMap* m, const void* base, int64_t rows, int d, int box_rows) {
  tc_encode_fn enc = tc_get_encode();
  if (!enc) return false;
  cuuint64_t gdim[2] = {(cuuint64_t)d, (cuuint64_t)rows};
  cuuint64_t gstr[1] = {(cuuint64_t)d * 2};
  cuuint32_t box[2] = {64u, (cuuint32_t)box_rows};
  cuuint32_t estr[2] = {1u, 1u};
  return enc(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
             CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

struct TcHeads { float* part; float* m; float bias, tau; };   // NEXT-2 riding the score kernel (Rm = the weight rows W[64, d])

// returns 0 on success, 1 if the cooperative launch is not possible on this device / partition (nothing was enqueued),
// -1 on a CUDA / driver error (cudaGetLastError holds the code when it is a launch error).
// `q_ready`: two zero-initialised 64-bit words owned by the plan (the kernel leaves them zero).
// `Rm` / `sig` (both NULL = off): NEXT-1, hash rows R[64, d] and the per-token signatures; requires every L <= 64.
// `hf` (NULL = off): NEXT-2, Rm = the head weight rows; same requirement; sig is ignored then.
inline int tc_launch_score(const TcSchedule& sc, const void* X, const void* Q, float* qinv, float* s, float* dnorm, float* rel,
                           unsigned long long* q_ready, int64_t N, int64_t nQ, int d, bool inline_qprep, const void* Rm, unsigned long long* sig,
                           const TcHeads* hf, cudaStream_t st, bool pdl_in = false) {
  TcMaps maps;
  for (int k = 0; k < 16; ++k)
    if (!tc_make_map(&maps.x[k], X, N, d, 16 * (k + 1))) return -1;
  for (int k = 0; k < 3; ++k)
    if (!tc_make_map(&maps.q[k], Q, nQ, d, 64 >> k)) return -1;
  if (sig != nullptr || hf != nullptr) { if (!tc_make_map(&maps.r, Rm, 64, d, 64)) return -1; } else maps.r = maps.q[0];
  TcParams p;
  p.tiles = sc.d_tiles; p.cta_off = sc.d_cta_off; p.qinv = qinv; p.Q = Q; p.nQ = nQ; p.q_ready = q_ready; p.sig = sig; p.s = s; p.dnorm = dnorm; p.rel = rel;
  p.d = d; p.n_kchunks = d / 64; p.roles_split = sc.roles_split ? 1 : 0;
#ifdef MSAS_ABLATE
  if (getenv("MSAS_ROLES")) p.roles_split = atoi(getenv("MSAS_ROLES"));
#endif
  p.heads_part = hf ? hf->part : nullptr; p.heads_m = hf ? hf->m : nullptr; p.heads_bias = hf ? hf->bias : 0.f; p.heads_tau = hf ? hf->tau : 0.f;
  if (hf) p.sig = nullptr;
#ifdef MSAS_ABLATE
  p.dbg = getenv("MSAS_ABLATE") ? atoi(getenv("MSAS_ABLATE")) : 0;
  static unsigned long long* dbuf = nullptr;
  if (!dbuf) cudaMalloc(&dbuf, 4096 * 8);
  p.dbg_t = dbuf;
#endif
  if (!inline_qprep) {   // qinv is already there: no CTA waits on another one, a plain launch will do
    p.Q = nullptr;
    if (launch_k(k_score_tc, dim3((unsigned)sc.n_ctas), dim3(kTcThreads), (size_t)sc.smem_bytes, st, pdl_in, maps, p) != cudaSuccess) return -1;
  } else {   // cooperative launch: the query-norm prologue makes the CTAs wait on one another once, so all must be resident
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)sc.n_ctas); cfg.blockDim = dim3(kTcThreads); cfg.dynamicSmemBytes = (size_t)sc.smem_bytes; cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeCooperative;
    attr[0].val.cooperative = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    const cudaError_t e = cudaLaunchKernelEx(&cfg, k_score_tc, maps, p);
    if (e == cudaErrorCooperativeLaunchTooLarge || e == cudaErrorNotSupported) return 1;   // caller: run k_qprep, then launch with inline_qprep = false
    if (e != cudaSuccess) return -1;
  }
#ifdef MSAS_ABLATE
  if (getenv("MSAS_TIMES")) {
    cudaStreamSynchronize(st);
    std::vector<unsigned long long> h(sc.n_ctas * 8);
    cudaMemcpy(h.data(), dbuf, h.size() * 8, cudaMemcpyDeviceToHost);
    unsigned long long t0 = ~0ull;
    for (int c = 0; c < sc.n_ctas; ++c) t0 = std::min(t0, h[c * 8]);
    if (getenv("MSAS_TIMES")[0] == '2')
      for (int c = 0; c < sc.n_ctas; ++c) fprintf(stderr, "cta %d sm %d end %.1f\n", c, (int)h[c * 8 + 1], (double)(h[c * 8 + 3] - t0) * 1e-3);
    {

    }
    {
      std::vector<unsigned long long> tt(128);
      cudaMemcpy(tt.data(), dbuf + 2048, 128 * 8, cudaMemcpyDeviceToHost);
      for (int b = 0; b < 2; ++b) { fprintf(stderr, "cta %d tile starts:", b ? 77 : 0); for (int i = 0; i < 12; ++i) fprintf(stderr, " %.1f", (double)(tt[b * 64 + i] - t0) * 1e-3); fprintf(stderr, "\n"); }
    }
    for (int k = 2; k < 4; ++k) {
      std::vector<double> v;
      for (int c = 0; c < sc.n_ctas; ++c) v.push_back((double)(h[c * 8 + k] - t0) * 1e-3);
      std::sort(v.begin(), v.end());
      fprintf(stderr, "stamp%d us: min %.1f p10 %.1f p50 %.1f p90 %.1f max %.1f\n", k, v[0], v[v.size() / 10], v[v.size() / 2],
              v[v.size() * 9 / 10], v.back());
    }
  }
#endif
  return cudaPeekAtLastError() == cudaSuccess ? 0 : -1;
}

}  // namespace msas
