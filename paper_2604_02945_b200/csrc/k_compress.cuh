// k_compress.cuh — NEXT-3, the rest of PAPER.md:98 / 105: spatial pooling of the scalar map (Eq. 3's AvgPool),
// one merged mean token per frame from the dropped rows ("coarsely compressed"), residual coding of kept video rows
// ("represented using only the residual difference").  All three are plain HBM / L2 streaming kernels.
#pragma once
#include "msas_internal.cuh"

namespace msas {

// One frame of the batch: its first row and its patch count (frames are numbered segment by segment).
struct DevFrame {
  int64_t row0;
  int32_t n_patches;
  int32_t seg;
};

// (a) k x k count-valid window mean of s on each frame's H x W grid; one thread per token (the map is 4 B per token: L2 resident).
__global__ void __launch_bounds__(256) k_spatial_pool(const DevSeg* __restrict__ segs, const DevTile* __restrict__ tiles,
                                                      const int32_t* __restrict__ grid_w, int k, const float* __restrict__ s,
                                                      float* __restrict__ out) {
  const DevTile tile = tiles[blockIdx.x];
  const DevSeg seg = segs[tile.seg];
  const int W = grid_w[tile.seg], H = seg.n_patches / W, lo = (k - 1) / 2, hi = k / 2;
  for (int r = threadIdx.x; r < tile.n_rows; r += blockDim.x) {
    const int64_t row = (int64_t)tile.row_start + r;
    const int64_t in_seg = row - seg.row0;
    const int t = (int)(in_seg / seg.n_patches), c = (int)(in_seg - (int64_t)t * seg.n_patches), i = c / W, j = c - i * W;
    const float* g = s + seg.row0 + (int64_t)t * seg.n_patches;
    float acc = 0.f;
    int cnt = 0;
    for (int a = max(i - lo, 0); a <= min(i + hi, H - 1); ++a)
      for (int b = max(j - lo, 0); b <= min(j + hi, W - 1); ++b) { acc += g[a * W + b]; ++cnt; }
    out[row] = acc / (float)cnt;
  }
}

// (b) mean of a frame's dropped rows.  One CTA of four warps per (frame, slab of 128 16-byte column vectors, row split); consecutive
// CTAs take the slabs of one frame.  Each warp takes every 4th row of its row range: the mask bytes of 32 rows at once, then only the
// dropped rows, four at a time (16 vector loads per lane), lanes cover the slab's vectors; fp32 sums in a fixed order.  With one row
// split the CTA writes the mean; with several (few frames: a batch of images) it writes partial sums and k_merge_finish adds them in
// split order.
constexpr int kMergeCtas = 1184;                 // CTAs aimed at when a batch has few frames (8 per SM); also the scratch slabs
constexpr int kMergeVPL = 4;                     // vectors per lane: a slab is 32 lanes x 4 vectors
constexpr int kMergeWarps = 4;                   // warps per CTA: small CTAs, so that a video batch's (frame, slab) units are all resident at once
template <int DT>
__global__ void __launch_bounds__(32 * kMergeWarps) k_merge_dropped(const DevFrame* __restrict__ frames, const void* __restrict__ X,
                                                       const uint8_t* __restrict__ keep_mask, float* __restrict__ Ymerge,
                                                       int32_t* __restrict__ n_dropped, float* __restrict__ part,
                                                       int32_t* __restrict__ cnt_part, int d) {
  constexpr int VE = DT == 1 ? 8 : 4;            // elements per 16-byte vector
  constexpr int VPL = kMergeVPL;
  constexpr int SLAB = 32 * VPL * VE;            // columns per slab
  constexpr int NW = kMergeWarps;
  __shared__ float red[NW][32 * VE];              // [warp][one vector index of the slab]
  __shared__ int cnt_s[NW];
  // consecutive CTAs take the slabs of ONE frame (the CTAs that run side by side read neighbouring pieces of the same rows)
  const unsigned lin = blockIdx.x + gridDim.x * blockIdx.y;
  const int fidx = (int)(lin / gridDim.y), sidx = (int)(lin % gridDim.y);
  const DevFrame fr = frames[fidx];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int RS = gridDim.z, rs = blockIdx.z;
  const int per = (fr.n_patches + RS - 1) / RS, p_lo = min(fr.n_patches, rs * per), p_hi = min(fr.n_patches, p_lo + per);
  const int c0 = sidx * SLAB;
  const int esz = DT == 1 ? 2 : 4;
  float acc[VPL][VE];
#pragma unroll
  for (int v = 0; v < VPL; ++v)
#pragma unroll
    for (int e = 0; e < VE; ++e) acc[v][e] = 0.f;
  int cnt = 0;
  // This warp's rows are p_lo + warp + NW j.  The mask bytes of 32 of them are read at once (one per lane) and turned into a bit mask
  // of the DROPPED ones; the loads then visit only those, four rows (16 vector loads per lane) at a time, in ascending order: the
  // mask latency is off the load chain and kept rows take no load slots.  (Same summation order as a plain row loop.)
  const int nj = p_hi > p_lo + warp ? (p_hi - p_lo - warp + NW - 1) / NW : 0;
  for (int j0 = 0; j0 < nj; j0 += 32) {
    const int prl = p_lo + warp + NW * (j0 + lane);
    unsigned m = __ballot_sync(0xffffffffu, prl < p_hi && keep_mask[fr.row0 + prl] == 0);
    cnt += __popc(m);
    while (m) {
      int pr[4];
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        if (m) { const int b = __ffs(m) - 1; m &= m - 1; pr[q] = p_lo + warp + NW * (j0 + b); } else pr[q] = -1;
      }
      uint4 u[4][VPL];
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const char* src = static_cast<const char*>(X) + (fr.row0 + (pr[q] < 0 ? 0 : pr[q])) * (int64_t)d * esz;
#pragma unroll
        for (int v = 0; v < VPL; ++v) {
          const int col = c0 + (v * 32 + lane) * VE;
          u[q][v] = (pr[q] >= 0 && col < d) ? ld_nc16(src + (int64_t)col * esz) : make_uint4(0, 0, 0, 0);
        }
      }
#pragma unroll
      for (int q = 0; q < 4; ++q) {
#pragma unroll
        for (int v = 0; v < VPL; ++v) {
          if (DT == 1) {
            const uint32_t w[4] = {u[q][v].x, u[q][v].y, u[q][v].z, u[q][v].w};
#pragma unroll
            for (int k = 0; k < 4; ++k) { acc[v][(2 * k) % VE] += bf_lo(w[k]); acc[v][(2 * k + 1) % VE] += bf_hi(w[k]); }
          } else {
            acc[v][0] += __uint_as_float(u[q][v].x); acc[v][1] += __uint_as_float(u[q][v].y);
            acc[v][2 % VE] += __uint_as_float(u[q][v].z); acc[v][3 % VE] += __uint_as_float(u[q][v].w);
          }
        }
      }
    }
  }
  if (lane == 0) cnt_s[warp] = cnt;
  __syncthreads();
  int total = 0;
#pragma unroll
  for (int w = 0; w < NW; ++w) total += cnt_s[w];
  const bool final_ = RS == 1;
  const float scale = final_ ? (total > 0 ? 1.0f / (float)total : 0.f) : 1.0f;
  if (sidx == 0 && threadIdx.x == 0) {
    if (final_) n_dropped[fidx] = total; else cnt_part[fidx * RS + rs] = total;
  }
  float* dst = final_ ? Ymerge + (int64_t)fidx * d : part + ((int64_t)(fidx * RS + rs) * gridDim.y + sidx) * SLAB - c0;
#pragma unroll
  for (int v = 0; v < VPL; ++v) {
    __syncthreads();
#pragma unroll
    for (int e = 0; e < VE; ++e) red[warp][lane * VE + e] = acc[v][e];
    __syncthreads();
    for (int i = threadIdx.x; i < 32 * VE; i += 32 * NW) {
      float t = 0.f;
#pragma unroll
      for (int w = 0; w < NW; ++w) t += red[w][i];
      const int col = c0 + v * 32 * VE + i;   // i = lane * VE + e
      if (col < d) dst[col] = t * scale;
    }
  }
}
// adds the row splits' partial sums in split order: one CTA per (frame, slab)
__global__ void __launch_bounds__(256) k_merge_finish(const float* __restrict__ part, const int32_t* __restrict__ cnt_part,
                                                      float* __restrict__ Ymerge, int32_t* __restrict__ n_dropped, int RS, int slab, int d) {
  const int f = blockIdx.x, y = blockIdx.y;
  int total = 0;
  for (int r = 0; r < RS; ++r) total += cnt_part[f * RS + r];
  if (y == 0 && threadIdx.x == 0) n_dropped[f] = total;
  const float inv = total > 0 ? 1.0f / (float)total : 0.f;
  for (int i = threadIdx.x; i < slab; i += 256) {
    const int col = y * slab + i;
    if (col >= d) break;
    float t = 0.f;
    for (int r = 0; r < RS; ++r) t += part[((int64_t)(f * RS + r) * gridDim.y + y) * slab + i];
    Ymerge[(int64_t)f * d + col] = t * inv;
  }
}

// (b') the same through the TMA unit, for rows of at most 16 KB.  LSU loads stream the dropped rows at about 4 TB/s; bulk copies
// into shared memory reach the HBM rate.  Persistent CTAs, one per SM: CTA c owns the global rows [c R, (c + 1) R) -- frames tile
// the rows in order, so it sees a run of frames, the first and the last possibly shared with its neighbours.  One producer warp
// reads the mask bytes of 32 rows at a time and issues one bulk copy (cp.async.bulk, mbarrier complete_tx) per DROPPED row into a
// ring of row slots; eight consumer warps each own an eighth of the row's 16-byte vectors and add them to fp32 accumulators in
// ascending row order (they read the same mask bytes, so they know which rows arrive).  A frame that lies inside one CTA's rows
// is written as its mean at once; a piece of a frame shared with a neighbour goes to slot 2c (the frame began before this
// CTA's rows) or 2c + 1 (it continues beyond them) of the scratch, and k_merge_tma_finish adds a frame's pieces in CTA order.
constexpr int kMergeTmaWarps = 8;                // consumer warps
constexpr int kMergeTmaVPL = 4;                  // 16-byte vectors per lane at most: rows of <= 8 * 32 * 4 * 16 B = 16 KB
constexpr int kMergeTmaSmem = 200 * 1024;        // ring bytes at most
__device__ __forceinline__ void bulk_load(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar, uint64_t pol) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(dst), "l"(src),
               "r"(bytes), "r"(bar), "l"(pol)
               : "memory");
}
__device__ __forceinline__ void add_f32x2(uint64_t& acc, uint64_t a) { asm("add.rn.f32x2 %0, %0, %1;" : "+l"(acc) : "l"(a)); }
template <int DT, int VPL>   // VPL: 16-byte vectors of a row per lane (1, 2 or 4)
__global__ void __launch_bounds__(32 * (kMergeTmaWarps + 1), 1)
k_merge_tma(const DevFrame* __restrict__ frames, int n_frames, const char* __restrict__ X, const uint8_t* __restrict__ keep_mask,
            float* __restrict__ Ymerge, int32_t* __restrict__ n_dropped, float* __restrict__ part, int32_t* __restrict__ cnt_part, int d,
            long long N, long long R, int n_slots) {
  constexpr int VE = DT == 1 ? 8 : 4;
  constexpr int NW = kMergeTmaWarps;
  extern __shared__ unsigned char merge_smem_raw[];
  unsigned char* smem = reinterpret_cast<unsigned char*>((reinterpret_cast<uintptr_t>(merge_smem_raw) + 127) & ~(uintptr_t)127);
  uint64_t* full = reinterpret_cast<uint64_t*>(smem);          // [n_slots] producer -> consumers (1 arrival + row bytes)
  uint64_t* empty = full + 32;                                  // [n_slots] consumers -> producer (NW arrivals)
  const uint32_t ring = smem_u32(smem) + 512u;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t row_bytes = (uint32_t)d * (DT == 1 ? 2u : 4u);
  const int n16 = (int)(row_bytes >> 4);                        // 16-byte vectors per row
  const int vpw = (n16 + NW - 1) / NW;                          // vectors per consumer warp
  if (threadIdx.x == 0) {
    for (int i = 0; i < n_slots; ++i) { mbar_init(smem_u32(&full[i]), 1); mbar_init(smem_u32(&empty[i]), NW); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  const long long lo = (long long)blockIdx.x * R, hi = lo + R < N ? lo + R : N;
  if (lo >= hi) return;
  int f = 0;                                                    // the frame that holds row `lo`
  { int a = 0, b = n_frames - 1; while (a < b) { const int m = (a + b + 1) >> 1; if (frames[m].row0 <= lo) a = m; else b = m - 1; } f = a; }
  uint32_t slot = 0, ph = 0;
  if (warp == NW) {
    // ---- producer
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    for (long long r0 = lo; r0 < hi; r0 += 32) {
      const long long r = r0 + lane;
      unsigned m = __ballot_sync(0xffffffffu, r < hi && keep_mask[r] == 0);
      while (m) {
        const int b = __ffs(m) - 1; m &= m - 1;
        mbar_wait(smem_u32(&empty[slot]), ph ^ 1u);
        if (lane == 0) {
          const uint32_t bar = smem_u32(&full[slot]);
          mbar_expect_tx(bar, row_bytes);
          bulk_load(ring + slot * row_bytes, X + (r0 + b) * (long long)row_bytes, row_bytes, bar, pol);
        }
        __syncwarp();
        if (++slot == (uint32_t)n_slots) { slot = 0; ph ^= 1u; }
      }
    }
    return;
  }
  // ---- consumers: warp w owns vectors [w vpw, (w + 1) vpw) of a row, lane l the vectors w vpw + l + 32 j
  // bf16: packed fp32 pairs (one FADD2 per two columns); fp32: plain adds
  uint64_t acc2[VPL][4];
  float acc[VPL][4];
  long long r = lo;
  while (r < hi) {
    const DevFrame fr = frames[f];
    const long long f_lo = fr.row0, f_hi = fr.row0 + fr.n_patches;
    const long long p_hi = f_hi < hi ? f_hi : hi;               // this CTA's piece of frame f: rows [r, p_hi)
#pragma unroll
    for (int j = 0; j < VPL; ++j)
#pragma unroll
      for (int e = 0; e < 4; ++e) { acc[j][e] = 0.f; acc2[j][e] = 0ull; }
    int cnt = 0;
    // the mask groups of the producer start at lo + 32 k: walk the piece group by group, masking off rows outside it
    for (long long g0 = lo + ((r - lo) & ~31ll); g0 < p_hi; g0 += 32) {
      const long long rr = g0 + lane;
      unsigned m = __ballot_sync(0xffffffffu, rr >= r && rr < p_hi && keep_mask[rr] == 0);
      cnt += __popc(m);
      for (int k = __popc(m); k > 0; --k) {
        mbar_wait(smem_u32(&full[slot]), ph);
        const uint32_t base = ring + slot * row_bytes;
        uint4 u[VPL];
        uint32_t seen = 0;
#pragma unroll
        for (int j = 0; j < VPL; ++j) {
          const int v = warp * vpw + lane + 32 * j;
          u[j] = (lane + 32 * j < vpw && v < n16) ? lds128(base + (uint32_t)v * 16u) : make_uint4(0, 0, 0, 0);
          seen |= u[j].x ^ u[j].w;
        }
        // the slot is released as soon as this warp's share of it is in registers (the empty asm consumes the loaded values, so
        // the arrive cannot be issued ahead of them)
        asm volatile("" ::"r"(seen) : "memory");
        __syncwarp();
        if (lane == 0) mbar_arrive(smem_u32(&empty[slot]));
#pragma unroll
        for (int j = 0; j < VPL; ++j) {
          if (DT == 1) {
            add_f32x2(acc2[j][0], bf16x2_to_f32x2(u[j].x)); add_f32x2(acc2[j][1], bf16x2_to_f32x2(u[j].y));
            add_f32x2(acc2[j][2], bf16x2_to_f32x2(u[j].z)); add_f32x2(acc2[j][3], bf16x2_to_f32x2(u[j].w));
          } else {
            acc[j][0] += __uint_as_float(u[j].x); acc[j][1] += __uint_as_float(u[j].y); acc[j][2] += __uint_as_float(u[j].z); acc[j][3] += __uint_as_float(u[j].w);
          }
        }
        if (++slot == (uint32_t)n_slots) { slot = 0; ph ^= 1u; }
      }
    }
    const bool whole = f_lo >= lo && f_hi <= hi;                // the frame lies inside this CTA's rows: write its mean
    const float scale = whole ? (cnt > 0 ? 1.0f / (float)cnt : 0.f) : 1.0f;
    const int pslot = 2 * (int)blockIdx.x + (f_lo < lo ? 0 : 1);
    float* dst = whole ? Ymerge + (long long)f * d : part + (long long)pslot * d;
    if (warp == 0 && lane == 0) { if (whole) n_dropped[f] = cnt; else cnt_part[pslot] = cnt; }
#pragma unroll
    for (int j = 0; j < VPL; ++j) {
      const int v = warp * vpw + lane + 32 * j;
      if (lane + 32 * j < vpw && v < n16) {
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          if (DT == 1) {
            float lo2, hi2;
            asm("mov.b64 {%0, %1}, %2;" : "=f"(lo2), "=f"(hi2) : "l"(acc2[j][e]));
            dst[v * VE + 2 * e] = lo2 * scale; dst[v * VE + 2 * e + 1] = hi2 * scale;
          } else {
            dst[v * VE + e] = acc[j][e] * scale;
          }
        }
      }
    }
    r = p_hi;
    ++f;
  }
}
// frames shared by several CTAs of k_merge_tma: their pieces added in CTA order; one CTA per frame (most return at once)
__global__ void __launch_bounds__(256) k_merge_tma_finish(const DevFrame* __restrict__ frames, const float* __restrict__ part,
                                                          const int32_t* __restrict__ cnt_part, float* __restrict__ Ymerge,
                                                          int32_t* __restrict__ n_dropped, int d, long long R) {
  const int f = blockIdx.x;
  const DevFrame fr = frames[f];
  const long long c0 = fr.row0 / R, c1 = (fr.row0 + fr.n_patches - 1) / R;
  if (c0 == c1) return;
  int total = 0;
  for (long long c = c0; c <= c1; ++c) total += cnt_part[2 * c + (fr.row0 < c * R ? 0 : 1)];
  if (threadIdx.x == 0) n_dropped[f] = total;
  const float inv = total > 0 ? 1.0f / (float)total : 0.f;
  // d % 4 == 0 (16-byte rows); the scratch slots are d floats apart and 16-byte aligned
  for (int i = threadIdx.x * 4; i < d; i += 1024) {
    float4 t = make_float4(0.f, 0.f, 0.f, 0.f);
    for (long long c = c0; c <= c1; ++c) {
      const float4 v = *reinterpret_cast<const float4*>(part + (2 * c + (fr.row0 < c * R ? 0 : 1)) * (long long)d + i);
      t.x += v.x; t.y += v.y; t.z += v.z; t.w += v.w;
    }
    float* y = Ymerge + (long long)f * d + i;
    y[0] = t.x * inv; y[1] = t.y * inv; y[2] = t.z * inv; y[3] = t.w * inv;
  }
}

// (c) gather with residual coding: kept row j of a temporal segment's frame t >= 1 is written as x_t - x_{t-1}; one warp per row.
template <int DT>
__global__ void __launch_bounds__(256) k_gather_residual(const DevSeg* __restrict__ segs, int n_segs, const char* __restrict__ X,
                                                         char* __restrict__ Y, const int32_t* __restrict__ kept_idx,
                                                         const int64_t* __restrict__ total_ptr, int64_t cap_rows, int d) {
  const int lane = threadIdx.x & 31;
  const int64_t total = *total_ptr < cap_rows ? *total_ptr : cap_rows;
  const int64_t n_warps = (int64_t)gridDim.x * 8;
  const int esz = DT == 1 ? 2 : 4;
  const int n16 = (d * esz) >> 4;
  for (int64_t j = (int64_t)blockIdx.x * 8 + (threadIdx.x >> 5); j < total; j += n_warps) {
    const int64_t row = kept_idx[j];
    int lo = 0, hi = n_segs - 1;               // the segment holding `row` (segments tile [0, N) in order)
    while (lo < hi) { const int mid = (lo + hi + 1) >> 1; if (segs[mid].row0 <= row) lo = mid; else hi = mid - 1; }
    const DevSeg sg = segs[lo];
    const bool res = sg.n_frames > 1 && row - sg.row0 >= sg.n_patches;
    const uint4* src = reinterpret_cast<const uint4*>(X + row * (int64_t)d * esz);
    const uint4* prv = reinterpret_cast<const uint4*>(X + (row - sg.n_patches) * (int64_t)d * esz);
    uint4* dst = reinterpret_cast<uint4*>(Y + j * (int64_t)d * esz);
    auto diff = [&](uint4 v, const uint4& q) {
      if (DT == 1) {   // the difference of two bf16 values is exact in fp32; cvt.rn rounds it to nearest even
        v.x = pack_bf16x2(bf_lo(v.x) - bf_lo(q.x), bf_hi(v.x) - bf_hi(q.x));
        v.y = pack_bf16x2(bf_lo(v.y) - bf_lo(q.y), bf_hi(v.y) - bf_hi(q.y));
        v.z = pack_bf16x2(bf_lo(v.z) - bf_lo(q.z), bf_hi(v.z) - bf_hi(q.z));
        v.w = pack_bf16x2(bf_lo(v.w) - bf_lo(q.w), bf_hi(v.w) - bf_hi(q.w));
      } else {
        v.x = __float_as_uint(__uint_as_float(v.x) - __uint_as_float(q.x)); v.y = __float_as_uint(__uint_as_float(v.y) - __uint_as_float(q.y));
        v.z = __float_as_uint(__uint_as_float(v.z) - __uint_as_float(q.z)); v.w = __float_as_uint(__uint_as_float(v.w) - __uint_as_float(q.w));
      }
      return v;
    };
    // four vectors of the row (and of its predecessor) in flight per lane
    for (int i0 = lane; i0 < n16; i0 += 128) {
      uint4 v[4], q[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int i = i0 + 32 * u;
        v[u] = i < n16 ? ld_nc16(src + i) : make_uint4(0, 0, 0, 0);
        q[u] = res && i < n16 ? ld_nc16(prv + i) : make_uint4(0, 0, 0, 0);
      }
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int i = i0 + 32 * u;
        if (i < n16) st_na16(dst + i, res ? diff(v[u], q[u]) : v[u]);
      }
    }
  }
}

}  // namespace msas
