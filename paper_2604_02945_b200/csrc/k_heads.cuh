// k_heads.cuh — NEXT-2: the paper's learned heads with caller-supplied weights.
//   Eq. 3: M_i = sigmoid(w_sp . x_i + b_sp);  Eq. 4: rho;  Eq. 6: alpha_s = MLP([p ; z_s]),
//   p = mean of the request's query rows, z_s = mean of the segment's rows, one hidden ReLU layer; literal softmax
//   (PAPER.md:116); Eq. 7 with reading G8.
// The first layer is linear in z_s, so W1z . mean(x) = mean(W1z . x): the per-row projections ride the same tile kernel that
// computes w_sp . x (k_heads_proj, k_score_simple.cuh), which leaves per-tile column sums; nothing of size d is reduced here.
#pragma once
#include "../../include/msas.h"
#include "k_segment.cuh"
#include "msas_internal.cuh"

namespace msas {

constexpr int kHeadRows = MAS_HEADS_ROWS;   // 64

constexpr int kHeadSlabs = 8;               // column slabs of the p-half (grid.y of k_heads_q)

// cq[r][y][h] = (1 / L_r) sum over the columns of slab y of Wp[h][c] * sum_j Q[q0_r + j][c]  (the p-half of the first layer, in
// kHeadSlabs partial sums that k_heads_finish adds in slab order).  One CTA per (request, slab); the slab is walked in chunks of
// 64 16-byte vectors: the chunk's column sums of the request's query rows go to shared memory (4 row groups x 64 vectors,
// four loads in flight per thread), then warp w takes weight rows 8w..8w+7, two vectors per lane and row (16 loads in flight).
template <int DT>
__global__ void __launch_bounds__(256) k_heads_q(const void* __restrict__ Q, const void* __restrict__ Wp, const int32_t* __restrict__ req_seg_off,
                                                 const DevSeg* __restrict__ segs, float* __restrict__ cq, int d) {
  constexpr int VE = DT == 1 ? 8 : 4;          // elements per 16-byte vector
  constexpr int CH = 64 * VE;                  // columns per chunk
  __shared__ float qs[4][CH];
  __shared__ float qsum[CH];
  const int r = blockIdx.x, y = blockIdx.y, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int k0 = req_seg_off[r];
  if (k0 >= req_seg_off[r + 1]) return;   // a request without segments is never read
  const DevSeg seg = segs[k0];
  const int L = seg.L;
  const int cw = (((d + kHeadSlabs - 1) / kHeadSlabs) + VE - 1) / VE * VE;   // slab width, a whole number of vectors (d % VE == 0)
  const int c0 = min(d, y * cw), c1 = min(d, c0 + cw);
  auto unpack = [](const uint4& u, float (&f)[VE]) {
    if (DT == 1) {
      const uint32_t w[4] = {u.x, u.y, u.z, u.w};
#pragma unroll
      for (int k = 0; k < 4; ++k) { f[(2 * k) % VE] = bf_lo(w[k]); f[(2 * k + 1) % VE] = bf_hi(w[k]); }
    } else {
      f[0] = __uint_as_float(u.x); f[1] = __uint_as_float(u.y); f[2 % VE] = __uint_as_float(u.z); f[3 % VE] = __uint_as_float(u.w);
    }
  };
  const int esz = DT == 1 ? 2 : 4;
  const char* Qb = static_cast<const char*>(Q);
  const char* Wb = static_cast<const char*>(Wp);
  float racc[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) racc[i] = 0.f;
  for (int cb = c0; cb < c1; cb += CH) {
    {   // column sums of the query rows: vector v of the chunk, rows j = rg, rg + 4, ...
      const int v = tid & 63, rg = tid >> 6;
      const int col = cb + v * VE;
      float a[VE];
#pragma unroll
      for (int e = 0; e < VE; ++e) a[e] = 0.f;
      if (col < c1) {
        int jq = rg;
        for (; jq + 12 < L; jq += 16) {
          uint4 u[4];
#pragma unroll
          for (int k = 0; k < 4; ++k) u[k] = ld_nc16(Qb + ((int64_t)(seg.q0 + jq + 4 * k) * d + col) * esz);
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            float f[VE];
            unpack(u[k], f);
#pragma unroll
            for (int e = 0; e < VE; ++e) a[e] += f[e];
          }
        }
        for (; jq < L; jq += 4) {
          float f[VE];
          unpack(ld_nc16(Qb + ((int64_t)(seg.q0 + jq) * d + col) * esz), f);
#pragma unroll
          for (int e = 0; e < VE; ++e) a[e] += f[e];
        }
      }
#pragma unroll
      for (int e = 0; e < VE; ++e) qs[rg][v * VE + e] = a[e];
    }
    __syncthreads();
    for (int e = tid; e < CH; e += 256) qsum[e] = (qs[0][e] + qs[1][e]) + (qs[2][e] + qs[3][e]);
    __syncthreads();
    {   // weight rows 8 * warp .. 8 * warp + 7, vectors lane and lane + 32 of the chunk
      uint4 u[8][2];
#pragma unroll
      for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int k = 0; k < 2; ++k) {
          const int col = cb + (lane + 32 * k) * VE;
          u[i][k] = col < c1 ? ld_nc16(Wb + ((int64_t)(warp * 8 + i) * d + col) * esz) : make_uint4(0, 0, 0, 0);
        }
#pragma unroll
      for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int k = 0; k < 2; ++k) {
          float f[VE];
          unpack(u[i][k], f);
#pragma unroll
          for (int e = 0; e < VE; ++e) racc[i] = fmaf(f[e], qsum[(lane + 32 * k) * VE + e], racc[i]);
        }
    }
    __syncthreads();   // qs / qsum are rewritten by the next chunk
  }
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const float t = warp_sum(racc[i]);
    if (lane == 0) cq[((int64_t)r * kHeadSlabs + y) * kHeadRows + warp * 8 + i] = t / (float)L;
  }
}

struct HeadsArgs {
  const DevSeg* segs;
  const int32_t* req_seg_off;
  int n_segs, n_requests, tile_rows, hidden;
  DevParams prm;
  const float* part;      // [slots, 64] partial column sums: one slot per generic tile (k_heads_proj) or per block of a tcgen05 tile (k_score_tc)
  const int32_t* slot_rank;   // NULL: the segment's slots are its generic tiles; else [n_segs + 1] first slot of every segment
  const float* cq;        // [n_requests, kHeadSlabs, 64] from k_heads_q
  const float* gamma;     // [N] (may be NULL when no segment is temporal)
  const float* b1;        // [64]
  const float* w2;        // [64]
  float b2;
  mas_segment_out* seg_out;
  unsigned int* done_counter;
};

// One CTA per segment: per-tile partials summed in tile order (double), gamma_avg, the hidden layer, alpha; the last CTA
// does the per-request softmax and Eq. 7.
__global__ void __launch_bounds__(1024) k_heads_finish(HeadsArgs a) {
  __shared__ SegSmem sm;
  __shared__ double colsum[kHeadRows];
  __shared__ double colpart[16][kHeadRows];
  const int tid = threadIdx.x, NT = blockDim.x, NG = NT >> 6;   // 256 or 1024 threads (host: from the longest segment)
  pdl_wait();
  const int sidx = blockIdx.x;
  const DevSeg seg = a.segs[sidx];
  const int n = seg.n_rows;
  const int slot_lo = a.slot_rank ? a.slot_rank[sidx] : seg.tile0;
  const int slot_hi = a.slot_rank ? a.slot_rank[sidx + 1] : seg.tile0 + (n + a.tile_rows - 1) / a.tile_rows;
  {   // column c = tid % 64; the four thread groups take every fourth slot, four loads in flight each: a fixed summation tree
    const int c = tid & 63, grp = tid >> 6;
    double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
    int t = slot_lo + grp;
    for (; t + 3 * NG < slot_hi; t += 4 * NG) {
      const float v0 = a.part[(int64_t)t * kHeadRows + c], v1 = a.part[(int64_t)(t + NG) * kHeadRows + c];
      const float v2 = a.part[(int64_t)(t + 2 * NG) * kHeadRows + c], v3 = a.part[(int64_t)(t + 3 * NG) * kHeadRows + c];
      s0 += (double)v0; s1 += (double)v1; s2 += (double)v2; s3 += (double)v3;
    }
    for (; t < slot_hi; t += NG) s0 += (double)a.part[(int64_t)t * kHeadRows + c];
    colpart[grp][c] = (s0 + s1) + (s2 + s3);
  }
  __syncthreads();
  if (tid < kHeadRows) {
    double s = 0.0;
    for (int gq = 0; gq < NG; ++gq) s += colpart[gq][tid];
    colsum[tid] = s;
  }
  double gs = 0.0, d1 = 0.0, d2 = 0.0;
  const bool temporal = seg.n_frames > 1;
  if (temporal)
    for (int i = seg.n_patches + tid; i < n; i += NT) gs += (double)a.gamma[seg.row0 + i];
  block_sum3(sm, gs, d1, d2);   // its barriers also publish colsum
  double contrib = 0.0;
  if (tid >= 1 && tid <= a.hidden) {   // the hidden unit in double: its <= 63 products are free next to the reductions above
    double pq = 0.0;
#pragma unroll
    for (int y = 0; y < kHeadSlabs; ++y) pq += (double)a.cq[((int64_t)seg.request * kHeadSlabs + y) * kHeadRows + tid];
    const double pre = colsum[tid] / (double)n + pq + (double)a.b1[tid];
    contrib = (double)a.w2[tid] * fmax(pre, 0.0);
  }
  d1 = d2 = 0.0;
  block_sum3(sm, contrib, d1, d2);
  if (tid == 0) {
    mas_segment_out o;
    o.rho_spatial = (float)(colsum[0] / (double)n);
    o.gamma_avg = temporal ? (float)(gs / ((double)(seg.n_frames - 1) * (double)seg.n_patches)) : 0.f;
    o.alpha_mean = (float)(contrib + (double)a.b2);
    o.beta = 0.f; o.mas = 0.f; o.mean_s = 0.f; o.std_s = 0.f;
    o.n_tokens = n; o.n_kept = 0;
    a.seg_out[sidx] = o;
  }
  __threadfence();
  __syncthreads();
  if (tid == 0) sm.bcast[2] = (atomicAdd(a.done_counter, 1u) == (unsigned)a.n_segs - 1u) ? 1 : 0;
  __syncthreads();
  if (!sm.bcast[2]) return;
  __threadfence();
  volatile mas_segment_out* so = a.seg_out;
  const DevParams& p = a.prm;
  for (int r = tid; r < a.n_requests; r += NT) {
    const int k0 = a.req_seg_off[r], k1 = a.req_seg_off[r + 1];
    double mx = -INFINITY;
    for (int k = k0; k < k1; ++k) mx = fmax(mx, (double)so[k].alpha_mean);
    double zsum = 0.0;
    for (int k = k0; k < k1; ++k) zsum += exp((double)so[k].alpha_mean - mx);
    for (int k = k0; k < k1; ++k) {   // literal softmax and Eq. 7 in double: a few segments per request
      const double beta = exp((double)so[k].alpha_mean - mx) / zsum;
      const double at = a.segs[k].n_frames > 1 ? (double)p.lambda_temp : 0.0;
      so[k].beta = (float)beta;
      so[k].mas = (float)(1.0 - beta * (1.0 - (double)p.lambda_spatial * (double)so[k].rho_spatial - at * (1.0 - (double)so[k].gamma_avg)));
    }
  }
  if (tid == 0) *a.done_counter = 0u;
}

}  // namespace msas
