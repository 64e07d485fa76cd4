// k_score_tc.cuh — the Blackwell fast path of the score pass (SURVEY.md §8(a) rows a1+a2+a3 in ONE sweep over X),
// bf16 inputs with d % 64 == 0.
//
//   TMA (cp.async.bulk.tensor, SWIZZLE_128B) stages, per 64-column K-chunk, the token tile X[rows, kc], the matching
//   previous-frame tile X[rows - P, kc] (temporal segments only; an L2 hit, never a second HBM read) and the request's
//   query chunk Q[L, kc] into a multi-stage shared-memory ring.
//   One elected thread issues tcgen05.mma (kind::f16, bf16 x bf16 -> fp32, M = 128, N = pad16(L), K = 16) accumulating
//   S = X·Q^T in TMEM (two accumulators: the epilogue of tile i overlaps the MMAs of tile i+1).          (Eq. 6)
//   Eight CUDA-core warps read the same shared-memory tiles (conflict-free thanks to the hardware swizzle) and
//   accumulate sum x^2, sum (x - x_prev)^2, sum x_prev^2 in fp32.                                        (Eq. 3, Eq. 5)
//   Four epilogue warps read the accumulator rows with tcgen05.ld (one token row per thread, so the max over query
//   tokens needs no shuffles), scale by 1/|q_j| and 1/|x_i| and write s, gamma, rel: 12 B per token.
//
// Persistent: one CTA per SM walks a host-built, cost-balanced (LPT) tile list.  Tiles never straddle a segment.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <cstring>
#include <queue>
#include <vector>

#include "../../include/msas.h"
#include "msas_internal.cuh"

namespace msas {

struct TcTile {            // 32 bytes
  int32_t row_start;       // global row id of the first row
  int32_t n_rows;          // valid rows, <= box rows
  int32_t box_kind;        // 0: 128-row TMA box, 1: 64, 2: 32, 3: 16
  int32_t q_row0;          // first query row of the request
  int32_t L;               // query tokens of the request
  int32_t prev_delta;      // P if the segment is temporal (T > 1), else 0
  int32_t key_rows;        // leading rows of the tile that belong to frame 0 (gamma = 1)
  int32_t pad_;
};

constexpr int kTcThreads = 512;
constexpr int kTcMaxStages = 10;
constexpr int kTcBoxBytes = 128 * 128;    // 128 rows x 64 bf16 columns

struct TcSchedule {
  bool enabled = false;
  bool any_temporal = false;
  int n_ctas = 0, n_tiles = 0, stages = 0, lmax_pad = 16;
  int stage_bytes = 0, smem_bytes = 0;
  const TcTile* d_tiles = nullptr;
  const int32_t* d_cta_off = nullptr;
};

struct TcParams {
  const TcTile* tiles;
  const int32_t* cta_off;
  const float* qinv;
  float* s;
  float* gamma;
  float* rel;
  int d;
  int n_kchunks;
  int stages;
  int stage_bytes;
  int prev_off;       // byte offset of the previous-frame tile inside a stage (0 = no such region)
  int q_off;          // byte offset of the query chunk inside a stage
};

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
  uint64_t full[kTcMaxStages];       // TMA -> consumers           (1 arrival + transaction bytes)
  uint64_t empty[kTcMaxStages];      // consumers -> TMA           (1 MMA commit + 8 ALU warps)
  uint64_t tmem_full[2];             // MMA -> epilogue            (1 commit)
  uint64_t tmem_empty[2];            // epilogue -> MMA            (4 warps)
  uint64_t stat_full[2];             // ALU -> epilogue            (8 warps)
  uint64_t stat_empty[2];            // epilogue -> ALU            (4 warps)
  uint32_t tmem_base;
  uint32_t pad_[31];
  float rowstat[2][3][128];          // n2, D, n2_prev per tile row, double buffered
};
constexpr int kTcCtrlBytes = 4096;
static_assert(sizeof(TcCtrl) <= kTcCtrlBytes, "control block too large");

__device__ __forceinline__ int tc_box_rows(int kind) { return 128 >> kind; }

__global__ void __launch_bounds__(kTcThreads, 1)
k_score_tc(const __grid_constant__ CUtensorMap mx128, const __grid_constant__ CUtensorMap mx64, const __grid_constant__ CUtensorMap mx32,
           const __grid_constant__ CUtensorMap mx16, const __grid_constant__ CUtensorMap mq, const TcParams p) {
  extern __shared__ unsigned char smem_raw[];
  unsigned char* smem = reinterpret_cast<unsigned char*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  TcCtrl* ctrl = reinterpret_cast<TcCtrl*>(smem);
  unsigned char* stage0 = smem + kTcCtrlBytes;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int tile_lo = p.cta_off[blockIdx.x], tile_hi = p.cta_off[blockIdx.x + 1];
  const int S = p.stages, nk = p.n_kchunks;

  if (warp == 1 && lane == 0) {
    for (int i = 0; i < S; ++i) { mbar_init(smem_u32(&ctrl->full[i]), 1); mbar_init(smem_u32(&ctrl->empty[i]), 9); }
    for (int i = 0; i < 2; ++i) {
      mbar_init(smem_u32(&ctrl->tmem_full[i]), 1); mbar_init(smem_u32(&ctrl->tmem_empty[i]), 4);
      mbar_init(smem_u32(&ctrl->stat_full[i]), 8); mbar_init(smem_u32(&ctrl->stat_empty[i]), 4);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 2) {   // TMEM: 2 accumulators x 128 fp32 columns
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&ctrl->tmem_base)), "r"(256) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  if (warp == 0 && lane == 0) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(&mx128) : "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(&mx64) : "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(&mq) : "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = ctrl->tmem_base;

  if (warp == 0) {
    // ===================================================================== TMA producer (one thread)
    if (lane == 0) {
      int stage = 0; uint32_t phase = 0;
      for (int t = tile_lo; t < tile_hi; ++t) {
        const TcTile tile = p.tiles[t];
        const CUtensorMap* mx = tile.box_kind == 0 ? &mx128 : tile.box_kind == 1 ? &mx64 : tile.box_kind == 2 ? &mx32 : &mx16;
        const bool has_prev = tile.prev_delta > 0 && tile.key_rows < tile.n_rows;
        const int nqb = (tile.L + 15) >> 4;
        const uint32_t box_bytes = (uint32_t)tc_box_rows(tile.box_kind) * 128u;
        const uint32_t tx = box_bytes * (has_prev ? 2u : 1u) + (uint32_t)nqb * 2048u;
        for (int kc = 0; kc < nk; ++kc) {
          mbar_wait(smem_u32(&ctrl->empty[stage]), phase ^ 1u);
          const uint32_t bar = smem_u32(&ctrl->full[stage]);
          unsigned char* st = stage0 + (size_t)stage * p.stage_bytes;
          mbar_expect_tx(bar, tx);
          tma_load_2d(smem_u32(st), mx, bar, kc * 64, tile.row_start);
          if (has_prev) tma_load_2d(smem_u32(st + p.prev_off), mx, bar, kc * 64, tile.row_start - tile.prev_delta);
          for (int j = 0; j < nqb; ++j) tma_load_2d(smem_u32(st + p.q_off + j * 2048), &mq, bar, kc * 64, tile.q_row0 + 16 * j);
          if (++stage == S) { stage = 0; phase ^= 1u; }
        }
      }
    }
  } else if (warp == 1) {
    // ===================================================================== MMA issuer (one thread)
    if (lane == 0) {
      int stage = 0; uint32_t phase = 0;
      int it = 0;
      for (int t = tile_lo; t < tile_hi; ++t, ++it) {
        const int L = p.tiles[t].L;
        const int npad = ((L + 15) >> 4) << 4;
        const uint32_t idesc = umma_idesc_bf16(npad);
        const int acc = it & 1;
        const uint32_t acc_phase = (uint32_t)(it >> 1) & 1u;
        mbar_wait(smem_u32(&ctrl->tmem_empty[acc]), acc_phase ^ 1u);
        tc_fence_after();
        const uint32_t d_tmem = tmem_base + (uint32_t)acc * 128u;
        for (int kc = 0; kc < nk; ++kc) {
          mbar_wait(smem_u32(&ctrl->full[stage]), phase);
          tc_fence_after();
          unsigned char* st = stage0 + (size_t)stage * p.stage_bytes;
          const uint64_t adesc = umma_desc_sw128(smem_u32(st));
          const uint64_t bdesc = umma_desc_sw128(smem_u32(st + p.q_off));
#pragma unroll
          for (int k = 0; k < 4; ++k)   // 4 x K=16 inside the 128-byte swizzle atom: +32 B = +2 in the 16-byte address field
            tc_mma_bf16(d_tmem, adesc + (uint64_t)(2 * k), bdesc + (uint64_t)(2 * k), idesc, (uint32_t)(kc | k));
          tc_commit(smem_u32(&ctrl->empty[stage]));
          if (++stage == S) { stage = 0; phase ^= 1u; }
        }
        tc_commit(smem_u32(&ctrl->tmem_full[acc]));
      }
    }
  } else if (warp >= 4 && warp < 8) {
    // ===================================================================== epilogue: one accumulator row per thread
    const int q = warp - 4;                  // TMEM lane quarter this warp may access (warp % 4)
    const int r = q * 32 + lane;             // tile row
    int it = 0;
    for (int t = tile_lo; t < tile_hi; ++t, ++it) {
      const TcTile tile = p.tiles[t];
      const int acc = it & 1;
      const uint32_t ph = (uint32_t)(it >> 1) & 1u;
      const int nqb = (tile.L + 15) >> 4;
      const float* qinv = p.qinv + tile.q_row0;
      mbar_wait(smem_u32(&ctrl->tmem_full[acc]), ph);
      tc_fence_after();
      float m = -INFINITY;
      for (int cb = 0; cb < nqb; ++cb) {
        uint32_t v[16];
        tc_ld16(tmem_base + (uint32_t)acc * 128u + (uint32_t)cb * 16u + ((uint32_t)(q * 32) << 16), v);
        tc_wait_ld();
#pragma unroll
        for (int j = 0; j < 16; ++j) {
          const int col = cb * 16 + j;
          if (col < tile.L) m = fmaxf(m, __uint_as_float(v[j]) * __ldg(qinv + col));
        }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(smem_u32(&ctrl->tmem_empty[acc]));
      mbar_wait(smem_u32(&ctrl->stat_full[acc]), ph);
      const float n2 = ctrl->rowstat[acc][0][r], D = ctrl->rowstat[acc][1][r], n2p = ctrl->rowstat[acc][2][r];
      __syncwarp();
      if (lane == 0) mbar_arrive(smem_u32(&ctrl->stat_empty[acc]));
      if (r < tile.n_rows) {
        const int64_t row = (int64_t)tile.row_start + r;
        p.s[row] = sqrtf(n2 / (float)p.d);
        float g = 0.f;
        if (tile.prev_delta > 0) {
          if (r < tile.key_rows) g = 1.0f;
          else { const float den = sqrtf(n2) + sqrtf(n2p); g = den > 0.f ? sqrtf(D) / den : 0.f; }
        }
        p.gamma[row] = g;
        p.rel[row] = n2 > 0.f ? m / sqrtf(n2) : 0.f;
      }
    }
  } else if (warp >= 8) {
    // ===================================================================== CUDA-core statistics: two threads per tile row
    const int a = tid - 256;
    const int r = a >> 1, half = a & 1;
    int stage = 0; uint32_t phase = 0;
    int it = 0;
    for (int t = tile_lo; t < tile_hi; ++t, ++it) {
      const TcTile tile = p.tiles[t];
      const bool has_prev = tile.prev_delta > 0 && tile.key_rows < tile.n_rows;
      const bool active = r < tc_box_rows(tile.box_kind);
      float n2a = 0.f, n2b = 0.f, Da = 0.f, Db = 0.f, pa = 0.f, pb = 0.f;
      const uint32_t row_off = (uint32_t)r * 128u;
      for (int kc = 0; kc < nk; ++kc) {
        mbar_wait(smem_u32(&ctrl->full[stage]), phase);
        if (active) {
          const unsigned char* st = stage0 + (size_t)stage * p.stage_bytes;
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            const uint32_t off = row_off + ((uint32_t)((half * 4 + j) ^ (r & 7)) << 4);   // hardware 128-byte swizzle
            const uint4 x = *reinterpret_cast<const uint4*>(st + off);
            const uint32_t xw[4] = {x.x, x.y, x.z, x.w};
            if (has_prev) {
              const uint4 u = *reinterpret_cast<const uint4*>(st + p.prev_off + off);
              const uint32_t uw[4] = {u.x, u.y, u.z, u.w};
#pragma unroll
              for (int k = 0; k < 4; ++k) {
                const float x0 = bf_lo(xw[k]), x1 = bf_hi(xw[k]), u0 = bf_lo(uw[k]), u1 = bf_hi(uw[k]);
                n2a = fmaf(x0, x0, n2a); n2b = fmaf(x1, x1, n2b);
                pa = fmaf(u0, u0, pa); pb = fmaf(u1, u1, pb);
                const float e0 = x0 - u0, e1 = x1 - u1;
                Da = fmaf(e0, e0, Da); Db = fmaf(e1, e1, Db);
              }
            } else {
#pragma unroll
              for (int k = 0; k < 4; ++k) {
                const float x0 = bf_lo(xw[k]), x1 = bf_hi(xw[k]);
                n2a = fmaf(x0, x0, n2a); n2b = fmaf(x1, x1, n2b);
              }
            }
          }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(smem_u32(&ctrl->empty[stage]));
        if (++stage == S) { stage = 0; phase ^= 1u; }
      }
      float n2 = n2a + n2b, D = Da + Db, n2p = pa + pb;
      n2 += __shfl_xor_sync(0xffffffffu, n2, 1);
      D += __shfl_xor_sync(0xffffffffu, D, 1);
      n2p += __shfl_xor_sync(0xffffffffu, n2p, 1);
      const int buf = it & 1;
      const uint32_t ph = (uint32_t)(it >> 1) & 1u;
      mbar_wait(smem_u32(&ctrl->stat_empty[buf]), ph ^ 1u);
      if (half == 0) { ctrl->rowstat[buf][0][r] = n2; ctrl->rowstat[buf][1][r] = D; ctrl->rowstat[buf][2][r] = n2p; }
      __syncwarp();
      if (lane == 0) mbar_arrive(smem_u32(&ctrl->stat_full[buf]));
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 2) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(256) : "memory");
  }
}

// ------------------------------------------------------------------------------------------------ host side
// Tile decomposition of one segment: greedy TMA boxes of 128/64/32/16 rows (a last partial box of <16 valid rows).
inline int tc_count_tiles(int64_t n) {
  int c = 0;
  while (n >= 128) { n -= 128; ++c; }
  for (int b = 64; b >= 16; b >>= 1) if (n >= b) { n -= b; ++c; }
  return c + (n > 0 ? 1 : 0);
}
inline size_t tc_schedule_bytes(const mas_segment* segs, int32_t n_segs) {
  size_t tiles = 0;
  for (int32_t k = 0; k < n_segs; ++k) tiles += (size_t)tc_count_tiles((int64_t)segs[k].n_frames * segs[k].n_patches);
  return tiles * sizeof(TcTile) + 1024 * sizeof(int32_t) + 256;
}

// Builds the tile list (grouped per CTA) and the per-CTA offsets into `h_dst`; `d_dst` is where the image will live.
inline void tc_build_schedule(TcSchedule& sc, const mas_segment* segs, int32_t n_segs, const int64_t* q_off, int32_t d, int32_t dtype,
                              int sm_count, char* h_dst, char* d_dst) {
  sc = TcSchedule();
  if (dtype != MAS_BF16 || d % 64 != 0 || sm_count < 1 || sm_count > 1000) return;
  std::vector<TcTile> tiles;
  int lmax = 1;
  bool any_temporal = false;
  for (int32_t k = 0; k < n_segs; ++k) {
    const mas_segment& s = segs[k];
    const int64_t n = (int64_t)s.n_frames * s.n_patches;
    const int L = (int)(q_off[s.request + 1] - q_off[s.request]);
    lmax = std::max(lmax, L);
    const int P = s.n_frames > 1 ? s.n_patches : 0;
    any_temporal |= P > 0;
    int64_t r = 0;
    auto push = [&](int kind, int rows_valid) {
      TcTile t{};
      t.row_start = (int32_t)(s.row0 + r);
      t.n_rows = rows_valid;
      t.box_kind = kind;
      t.q_row0 = (int32_t)q_off[s.request];
      t.L = L;
      t.prev_delta = P;
      t.key_rows = P > 0 ? (int32_t)std::min<int64_t>(std::max<int64_t>(P - r, 0), rows_valid) : 0;
      tiles.push_back(t);
      r += rows_valid;
    };
    while (n - r >= 128) push(0, 128);
    for (int kind = 1; kind <= 3; ++kind) if (n - r >= (128 >> kind)) push(kind, 128 >> kind);
    if (n - r > 0) push(3, (int)(n - r));
  }
  const int n_tiles = (int)tiles.size();
  const int n_ctas = std::min(sm_count, n_tiles);
  // LPT: heaviest tile first onto the least-loaded CTA (ties -> lowest CTA id, which makes equal-cost tiles round-robin
  // in row order: neighbouring CTAs sweep neighbouring rows, so previous-frame tiles are still in L2).
  auto cost = [&](const TcTile& t) {
    const bool has_prev = t.prev_delta > 0 && t.key_rows < t.n_rows;
    return (int64_t)(128 >> t.box_kind) * (has_prev ? 2 : 1) + ((t.L + 15) / 16) * 16 + 8;
  };
  std::vector<int> order(n_tiles);
  for (int i = 0; i < n_tiles; ++i) order[i] = i;
  std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return cost(tiles[a]) > cost(tiles[b]); });
  typedef std::pair<int64_t, int> Load;   // (load, cta)
  std::priority_queue<Load, std::vector<Load>, std::greater<Load>> heap;
  for (int c = 0; c < n_ctas; ++c) heap.push(Load(0, c));
  std::vector<std::vector<int>> per(n_ctas);
  for (int i : order) {
    Load l = heap.top(); heap.pop();
    per[l.second].push_back(i);
    heap.push(Load(l.first + cost(tiles[i]), l.second));
  }
  TcTile* ht = reinterpret_cast<TcTile*>(h_dst);
  int32_t* hoff = reinterpret_cast<int32_t*>(h_dst + (size_t)n_tiles * sizeof(TcTile));
  int w = 0;
  for (int c = 0; c < n_ctas; ++c) {
    std::sort(per[c].begin(), per[c].end());   // ascending rows inside a CTA
    hoff[c] = w;
    for (int i : per[c]) ht[w++] = tiles[i];
  }
  hoff[n_ctas] = w;
  const int lmax_pad = ((lmax + 15) / 16) * 16;
  sc.any_temporal = any_temporal;
  sc.lmax_pad = lmax_pad;
  sc.stage_bytes = kTcBoxBytes * (any_temporal ? 2 : 1) + lmax_pad * 128;
  const int budget = 227 * 1024 - kTcCtrlBytes - 1024;
  sc.stages = std::min(kTcMaxStages, budget / sc.stage_bytes);
  if (sc.stages < 2) return;
  sc.smem_bytes = kTcCtrlBytes + 1024 + sc.stages * sc.stage_bytes;
  sc.n_ctas = n_ctas;
  sc.n_tiles = n_tiles;
  sc.d_tiles = reinterpret_cast<const TcTile*>(d_dst);
  sc.d_cta_off = reinterpret_cast<const int32_t*>(d_dst + (size_t)n_tiles * sizeof(TcTile));
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

// returns 0 on success, -1 on a CUDA / driver error (cudaGetLastError holds the code when it is a launch error)
inline int tc_launch_score(const TcSchedule& sc, const void* X, const void* Q, const float* qinv, float* s, float* gamma, float* rel,
                           int64_t N, int64_t nQ, int d, cudaStream_t st) {
  CUtensorMap mx[4], mq;
  for (int k = 0; k < 4; ++k)
    if (!tc_make_map(&mx[k], X, N, d, 128 >> k)) return -1;
  if (!tc_make_map(&mq, Q, nQ, d, 16)) return -1;
  TcParams p;
  p.tiles = sc.d_tiles; p.cta_off = sc.d_cta_off; p.qinv = qinv; p.s = s; p.gamma = gamma; p.rel = rel;
  p.d = d; p.n_kchunks = d / 64; p.stages = sc.stages; p.stage_bytes = sc.stage_bytes;
  p.prev_off = sc.any_temporal ? kTcBoxBytes : 0;
  p.q_off = kTcBoxBytes * (sc.any_temporal ? 2 : 1);
  k_score_tc<<<sc.n_ctas, kTcThreads, sc.smem_bytes, st>>>(mx[0], mx[1], mx[2], mx[3], mq, p);
  return cudaPeekAtLastError() == cudaSuccess ? 0 : -1;
}

}  // namespace msas
