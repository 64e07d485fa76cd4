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
// kHeadSlabs partial sums that k_heads_finish adds in slab order): one CTA per (request, slab), the slab's column sums of the
// request's query rows in shared memory, then one warp per weight row.
template <int DT>
__global__ void __launch_bounds__(256) k_heads_q(const void* __restrict__ Q, const void* __restrict__ Wp, const int32_t* __restrict__ req_seg_off,
                                                 const DevSeg* __restrict__ segs, float* __restrict__ cq, int d) {
  extern __shared__ float qsum[];
  const int r = blockIdx.x, y = blockIdx.y, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int k0 = req_seg_off[r];
  if (k0 >= req_seg_off[r + 1]) return;   // a request without segments is never read
  const DevSeg seg = segs[k0];
  const int L = seg.L;
  const int cw = (d + kHeadSlabs - 1) / kHeadSlabs, c0 = y * cw, c1 = min(d, c0 + cw);
  auto ld = [&](const void* base, int64_t at) {
    return DT == 1 ? __bfloat162float(static_cast<const __nv_bfloat16*>(base)[at]) : static_cast<const float*>(base)[at];
  };
  for (int col = c0 + threadIdx.x; col < c1; col += 256) {
    float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f;
    const int64_t at = (int64_t)seg.q0 * d + col;
    int j = 0;
    for (; j + 3 < L; j += 4) {
      a0 += ld(Q, at + (int64_t)j * d); a1 += ld(Q, at + (int64_t)(j + 1) * d);
      a2 += ld(Q, at + (int64_t)(j + 2) * d); a3 += ld(Q, at + (int64_t)(j + 3) * d);
    }
    for (; j < L; ++j) a0 += ld(Q, at + (int64_t)j * d);
    qsum[col - c0] = (a0 + a1) + (a2 + a3);
  }
  __syncthreads();
  for (int h = warp; h < kHeadRows; h += 8) {
    float a = 0.f;
    for (int col = c0 + lane; col < c1; col += 32) a = fmaf(ld(Wp, (int64_t)h * d + col), qsum[col - c0], a);
    a = warp_sum(a);
    if (lane == 0) cq[((int64_t)r * kHeadSlabs + y) * kHeadRows + h] = a / (float)L;
  }
}

struct HeadsArgs {
  const DevSeg* segs;
  const int32_t* req_seg_off;
  int n_segs, n_requests, tile_rows, hidden;
  DevParams prm;
  const float* part;      // [slots, 64] per-tile partials: generic tiles (k_heads_proj) or 2 halves per tcgen05 tile (k_score_tc)
  const int32_t* slot_rank;   // NULL: the segment's slots are its generic tiles; else [n_segs + 1] first tile rank per segment (x 2 halves)
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
__global__ void __launch_bounds__(256) k_heads_finish(HeadsArgs a) {
  __shared__ SegSmem sm;
  __shared__ double colsum[kHeadRows];
  const int tid = threadIdx.x;
  const int sidx = blockIdx.x;
  const DevSeg seg = a.segs[sidx];
  const int n = seg.n_rows;
  const int slot_lo = a.slot_rank ? 2 * a.slot_rank[sidx] : seg.tile0;
  const int slot_hi = a.slot_rank ? 2 * a.slot_rank[sidx + 1] : seg.tile0 + (n + a.tile_rows - 1) / a.tile_rows;
  if (tid < kHeadRows) {
    double s = 0.0;
    for (int t = slot_lo; t < slot_hi; ++t) s += (double)a.part[(int64_t)t * kHeadRows + tid];
    colsum[tid] = s;
  }
  double gs = 0.0, d1 = 0.0, d2 = 0.0;
  const bool temporal = seg.n_frames > 1;
  if (temporal)
    for (int i = seg.n_patches + tid; i < n; i += 256) gs += (double)a.gamma[seg.row0 + i];
  block_sum3(sm, gs, d1, d2);   // its barriers also publish colsum
  double contrib = 0.0;
  if (tid >= 1 && tid <= a.hidden) {
    float pq = 0.f;
#pragma unroll
    for (int y = 0; y < kHeadSlabs; ++y) pq += a.cq[((int64_t)seg.request * kHeadSlabs + y) * kHeadRows + tid];
    const float pre = (float)(colsum[tid] / (double)n) + pq + a.b1[tid];
    contrib = (double)(a.w2[tid] * fmaxf(pre, 0.f));
  }
  d1 = d2 = 0.0;
  block_sum3(sm, contrib, d1, d2);
  if (tid == 0) {
    mas_segment_out o;
    o.rho_spatial = (float)(colsum[0] / (double)n);
    o.gamma_avg = temporal ? (float)(gs / ((double)(seg.n_frames - 1) * (double)seg.n_patches)) : 0.f;
    o.alpha_mean = (float)contrib + a.b2;
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
  for (int r = tid; r < a.n_requests; r += 256) {
    const int k0 = a.req_seg_off[r], k1 = a.req_seg_off[r + 1];
    float mx = -INFINITY;
    for (int k = k0; k < k1; ++k) mx = fmaxf(mx, so[k].alpha_mean);
    float zsum = 0.f;
    for (int k = k0; k < k1; ++k) zsum += expf(so[k].alpha_mean - mx);
    for (int k = k0; k < k1; ++k) {
      const float beta = expf(so[k].alpha_mean - mx) / zsum;
      const float at = a.segs[k].n_frames > 1 ? p.lambda_temp : 0.f;
      so[k].beta = beta;
      so[k].mas = 1.0f - beta * (1.0f - p.lambda_spatial * so[k].rho_spatial - at * (1.0f - so[k].gamma_avg));
    }
  }
  if (tid == 0) *a.done_counter = 0u;
}

}  // namespace msas
