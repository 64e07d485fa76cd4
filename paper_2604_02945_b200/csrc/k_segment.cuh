// k_segment.cuh — K2: per-segment statistics, fusion and selection over the per-token scalars only
// and K3: the row gather (row a6).
//   a4  mean / population std of s and rel, M_i = sigma(z) (Eq. 3), rho (Eq. 4), gamma_avg, alpha, per-token MAS (SPEC S4),
//       then per request softmax -> beta and Eq. 7.
//   a5  exact k-th smallest (MAS_i, i) by 4 x 8-bit radix select on order-preserving keys, ties -> lower index;
//       or threshold MAS_i <= cut; warp ballot + block prefix scan -> kept_idx (ascending row ids).
//   a6  Y[j,:] = X[kept_idx[j],:], 16-byte copies, bit exact.
// All reductions are fixed-order (no floating-point atomics): runs are bit-reproducible.
#pragma once
#include "../../include/msas.h"
#include "msas_internal.cuh"

namespace msas {

struct SegArgs {
  const DevSeg* segs;
  const int32_t* req_seg_off;   // [R+1] first segment of each request
  int n_segs, n_requests;
  DevParams prm;
  const float* s;
  float* gamma;                 // FUSE: final gamma, or (gamma_raw) sqrt(D) from the tcgen05 score kernel, finished in place
  const float* rel;
  float* m_spatial;             // may be NULL
  float* mas_tok;               // FUSE: output; SELECT only: input
  mas_segment_out* seg_out;     // may be NULL
  uint8_t* keep_mask;           // may be NULL
  int32_t* kept_idx;            // may be NULL
  int64_t* kept_off;            // may be NULL
  int64_t cap_rows;
  int32_t* seg_nkept;           // workspace [n_segs]
  unsigned int* done_counter;   // workspace, zero between launches
  int gamma_raw;                // 1: gamma holds sqrt(sum (x_t - x_{t-1})^2); gamma = that / (|x_t| + |x_{t-1}|) (SPEC S2)
  float sqrt_d;                 // |x_i| = s_i * sqrt(d)
};

constexpr int kSegThreads = 1024;

struct SegSmem {
  double red[6][32];
  double tot[6];
  int ired[2][32];
  unsigned int hist[4][256];   // one histogram per radix pass (never reused or overwritten: peers read them over DSMEM)
  unsigned int htot[256];      // cluster-wide totals of the current pass
  int bcast[4];
  double cx_d[4][6];           // cluster exchange: this CTA's block totals of reduction round 0..3
  int cx_i[2];                 // cluster exchange: this CTA's (less, equal) counts
};

// ---- thread-block cluster helpers (a segment is shared by the CTAs of one cluster; cluster size 1 works too)
__device__ __forceinline__ unsigned cluster_rank() { unsigned r; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ unsigned cluster_size() { unsigned r; asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ unsigned cluster_id_x() { unsigned r; asm volatile("mov.u32 %0, %%clusterid.x;" : "=r"(r)); return r; }
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;\nbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
template <class T> __device__ __forceinline__ T dsmem_read(const T* local, unsigned rank);
template <> __device__ __forceinline__ double dsmem_read<double>(const double* local, unsigned rank) {
  unsigned a = (unsigned)__cvta_generic_to_shared(local), ra; double v;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(ra) : "r"(a), "r"(rank));
  asm volatile("ld.shared::cluster.f64 %0, [%1];" : "=d"(v) : "r"(ra) : "memory");
  return v;
}
template <> __device__ __forceinline__ int dsmem_read<int>(const int* local, unsigned rank) {
  unsigned a = (unsigned)__cvta_generic_to_shared(local), ra; int v;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(ra) : "r"(a), "r"(rank));
  asm volatile("ld.shared::cluster.b32 %0, [%1];" : "=r"(v) : "r"(ra) : "memory");
  return v;
}
template <> __device__ __forceinline__ unsigned dsmem_read<unsigned>(const unsigned* local, unsigned rank) {
  return (unsigned)dsmem_read<int>(reinterpret_cast<const int*>(local), rank);
}

// fixed-order block sum of up to three doubles (any block size that is a multiple of 32); result broadcast to every
// thread.  The second round runs in warp 0 only: double shuffles are two SHFLs each and 32 warps doing them again
// for the same 32 partials only queues up the shuffle pipe.
__device__ __forceinline__ void block_sum3(SegSmem& sm, double& a, double& b, double& c) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
  a = warp_sum(a); b = warp_sum(b); c = warp_sum(c);
  __syncthreads();
  if (lane == 0) { sm.red[0][warp] = a; sm.red[1][warp] = b; sm.red[2][warp] = c; }
  __syncthreads();
  if (warp == 0) {
    double x = lane < nw ? sm.red[0][lane] : 0.0, y = lane < nw ? sm.red[1][lane] : 0.0, z = lane < nw ? sm.red[2][lane] : 0.0;
    x = warp_sum(x); y = warp_sum(y); z = warp_sum(z);
    if (lane == 0) { sm.tot[0] = x; sm.tot[1] = y; sm.tot[2] = z; }
  }
  __syncthreads();
  a = sm.tot[0]; b = sm.tot[1]; c = sm.tot[2];
}

// exclusive prefix over the block of two small counts; also returns block totals
__device__ __forceinline__ void block_scan2(SegSmem& sm, int fa, int fb, int& pa, int& pb, int& ta, int& tb) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const unsigned ba = __ballot_sync(0xffffffffu, fa), bb = __ballot_sync(0xffffffffu, fb);
  const unsigned lt = (1u << lane) - 1u;
  __syncthreads();
  if (lane == 0) { sm.ired[0][warp] = __popc(ba); sm.ired[1][warp] = __popc(bb); }
  __syncthreads();
  const int nw = blockDim.x >> 5;
  int wa = lane < nw ? sm.ired[0][lane] : 0, wb = lane < nw ? sm.ired[1][lane] : 0;
  int ia = wa, ib = wb;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    int ua = __shfl_up_sync(0xffffffffu, ia, o), ub = __shfl_up_sync(0xffffffffu, ib, o);
    if (lane >= o) { ia += ua; ib += ub; }
  }
  ta = __shfl_sync(0xffffffffu, ia, 31);
  tb = __shfl_sync(0xffffffffu, ib, 31);
  const int ea = __shfl_sync(0xffffffffu, ia - wa, warp), eb = __shfl_sync(0xffffffffu, ib - wb, warp);
  pa = ea + __popc(ba & lt);
  pb = eb + __popc(bb & lt);
}

// fixed-order sum of up to three doubles over all CTAs of the cluster; the result reaches every thread of every CTA.
// `round` selects a private exchange slot (no slot is reused inside one launch, so one cluster barrier per round suffices).
__device__ __forceinline__ void cluster_sum3(SegSmem& sm, int round, unsigned nc, double& a, double& b, double& c) {
  block_sum3(sm, a, b, c);
  if (nc == 1) return;
  if (threadIdx.x == 0) { sm.cx_d[round][0] = a; sm.cx_d[round][1] = b; sm.cx_d[round][2] = c; }
  cluster_sync_all();
  // one lane per peer fetches its three totals (independent remote loads: one DSMEM latency, not 3 x nc of them)
  if (threadIdx.x < nc) {
    const double x = dsmem_read(&sm.cx_d[round][0], threadIdx.x), y = dsmem_read(&sm.cx_d[round][1], threadIdx.x),
                 z = dsmem_read(&sm.cx_d[round][2], threadIdx.x);
    sm.red[0][threadIdx.x] = x; sm.red[1][threadIdx.x] = y; sm.red[2][threadIdx.x] = z;
  }
  __syncthreads();
  double x = 0, y = 0, z = 0;
  for (unsigned r = 0; r < nc; ++r) { x += sm.red[0][r]; y += sm.red[1][r]; z += sm.red[2][r]; }   // rank order: same bits in every CTA
  a = x; b = y; c = z;
  __syncthreads();   // sm.red is reused by the next block_sum3
}

// six doubles at once (the one-pass segment statistics): same scheme, one block reduction and one cluster barrier
__device__ __forceinline__ void cluster_sum6(SegSmem& sm, int round, unsigned nc, double (&v)[6]) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
#pragma unroll
  for (int k = 0; k < 6; ++k) v[k] = warp_sum(v[k]);
  __syncthreads();
  if (lane == 0) {
#pragma unroll
    for (int k = 0; k < 6; ++k) sm.red[k][warp] = v[k];
  }
  __syncthreads();
  if (warp == 0) {
#pragma unroll
    for (int k = 0; k < 6; ++k) { const double x = warp_sum(lane < nw ? sm.red[k][lane] : 0.0); if (lane == 0) { sm.tot[k] = x; sm.cx_d[round][k] = x; } }
  }
  if (nc == 1) {
    __syncthreads();
#pragma unroll
    for (int k = 0; k < 6; ++k) v[k] = sm.tot[k];
    return;
  }
  cluster_sync_all();
  if (threadIdx.x < 6 * nc) sm.red[threadIdx.x % 6][threadIdx.x / 6] = dsmem_read(&sm.cx_d[round][threadIdx.x % 6], threadIdx.x / 6);
  __syncthreads();
#pragma unroll
  for (int k = 0; k < 6; ++k) { double x = 0; for (unsigned r = 0; r < nc; ++r) x += sm.red[k][r]; v[k] = x; }   // rank order
  __syncthreads();
}

// One thread-block CLUSTER per segment (cluster size chosen by the host from the longest segment; 1 for images):
// CTA `rank` owns the contiguous token slice [lo, hi) of the segment; sums, radix histograms and kept counts are
// combined over distributed shared memory, so an 18 432-token video segment is a few microseconds of latency, not 70.
template <bool FUSE, bool SELECT>
__global__ void __launch_bounds__(kSegThreads) k_segment(SegArgs a) {
  __shared__ SegSmem sm;
  const int NT = blockDim.x;      // 256, 512 or 1024 (host: from the longest per-CTA slice)
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const unsigned nc = cluster_size(), rank = cluster_rank();
  const int sidx = (int)cluster_id_x();
  const DevSeg seg = a.segs[sidx];
  const int n = seg.n_rows;
  const int64_t base = seg.row0;
  const DevParams& p = a.prm;
  const int per = (n + (int)nc - 1) / (int)nc;
  const int lo = min(n, (int)rank * per), hi = min(n, lo + per);
  pdl_launch_dependents();
  pdl_wait();

  constexpr int KPT = 4;          // tokens per thread whose scalars stay in registers between the passes
  float c_s[KPT], c_r[KPT], c_g[KPT];
  unsigned c_key[KPT];            // order-preserving keys of the cached tokens' MAS (selection passes)
#pragma unroll
  for (int it = 0; it < KPT; ++it) { c_s[it] = 0.f; c_r[it] = 0.f; c_g[it] = 0.f; c_key[it] = 0u; }

  if (FUSE) {
    const bool temporal = seg.n_frames > 1;
    // pass A: one sweep gives sum and sum of squares (double: the cancellation in E[x^2] - mu^2 is ~1e-14 relative
    // for these O(1) scalars); gamma is finished here (SPEC S2) because both norms are at hand
    auto load_token = [&](int i, float& si, float& ri, float& gi) {
      si = a.s[base + i];
      ri = a.rel[base + i];
      gi = 0.f;
      if (temporal) {
        if (a.gamma_raw) {
          if (i < seg.n_patches) gi = 1.0f;
          else { const float den = (si + a.s[base + i - seg.n_patches]) * a.sqrt_d; gi = den > 0.f ? a.gamma[base + i] / den : 0.f; }
        } else gi = a.gamma[base + i];
      }
      if (a.gamma_raw) a.gamma[base + i] = gi;
    };
    double acc[6] = {0, 0, 0, 0, 0, 0};   // sum s, sum s^2, sum r, sum r^2, sum gamma (t >= 1), unused
    auto accumulate = [&](int i, float si, float ri, float gi) {
      acc[0] += (double)si; acc[1] += (double)si * (double)si; acc[2] += (double)ri; acc[3] += (double)ri * (double)ri;
      if (temporal && i >= seg.n_patches) acc[4] += (double)gi;
    };
#pragma unroll
    for (int it = 0; it < KPT; ++it) {
      const int i = lo + tid + it * NT;
      if (i < hi) { load_token(i, c_s[it], c_r[it], c_g[it]); accumulate(i, c_s[it], c_r[it], c_g[it]); }
    }
    for (int i = lo + tid + KPT * NT; i < hi; i += NT) { float si, ri, gi; load_token(i, si, ri, gi); accumulate(i, si, ri, gi); }
    cluster_sum6(sm, 0, nc, acc);
    // one double division per thread (1 / n); the variances stay in double (E[x^2] - mu^2 cancels), everything after the
    // square root is needed to fp32 accuracy only (double division and sqrt are long software routines)
    const double inv_n = 1.0 / (double)n;
    const double mu_s = acc[0] * inv_n, mu_r = acc[2] * inv_n;
    const float gavg = temporal ? (float)acc[4] / ((float)(seg.n_frames - 1) * (float)seg.n_patches) : 0.f;
    const float sd_s = sqrtf((float)fmax(acc[1] * inv_n - mu_s * mu_s, 0.0)), sd_r = sqrtf((float)fmax(acc[3] * inv_n - mu_r * mu_r, 0.0));
    const float den_s = fmaxf(sd_s, 1e-6f * (float)mu_s), den_r = fmaxf(sd_r, 1e-6f);
    const float inv_s = den_s > 0.f ? 1.0f / den_s : 0.f, inv_r = 1.0f / den_r;
    const float at = temporal ? p.lambda_temp : 0.f;
    int below = 0;
    // pass B: per-token M, g, MAS (differences in double: the means are not representable in fp32)
    auto fuse_token = [&](int i, float si, float ri, float gi) {
      const float z = (float)(((double)si - mu_s)) * inv_s;
      const float M = sigmoidf_acc(p.spatial_gain * z + p.spatial_bias);
      const float zr = (float)(((double)ri - mu_r)) * inv_r;
      const float g = sigmoidf_acc(p.rel_gain * zr + p.rel_bias);
      const float mas = 1.0f - g * (1.0f - p.lambda_spatial * (1.0f - M) - at * (1.0f - gi));
      if (a.m_spatial) a.m_spatial[base + i] = M;
      a.mas_tok[base + i] = mas;
      below += M < p.tau_s ? 1 : 0;
      return mas;
    };
#pragma unroll
    for (int it = 0; it < KPT; ++it) {
      const int i = lo + tid + it * NT;
      if (i < hi) c_key[it] = float_key(fuse_token(i, c_s[it], c_r[it], c_g[it]));
    }
    for (int i = lo + tid + KPT * NT; i < hi; i += NT) {
      float si = a.s[base + i], ri = a.rel[base + i], gi = temporal ? a.gamma[base + i] : 0.f;
      fuse_token(i, si, ri, gi);
    }
    const float sd_s_out = sd_s;
    double db = below, d1 = 0, d2 = 0;
    cluster_sum3(sm, 2, nc, db, d1, d2);
    if (rank == 0 && tid == 0 && a.seg_out) {
      mas_segment_out o;
      o.rho_spatial = (float)(db / n);
      o.gamma_avg = gavg;
      o.alpha_mean = (float)mu_r;
      o.beta = 0.f; o.mas = 0.f;
      o.mean_s = (float)mu_s; o.std_s = sd_s_out;
      o.n_tokens = n; o.n_kept = 0;
      a.seg_out[sidx] = o;
    }
    __syncthreads();   // mas_tok of this CTA's slice is re-read below by other threads of the same CTA
  }

  if (SELECT) {
    const float* mas = a.mas_tok + base;
    if (!FUSE) {
#pragma unroll
      for (int it = 0; it < KPT; ++it) { const int i = lo + tid + it * NT; if (i < hi) c_key[it] = float_key(mas[i]); }
    }
    // visit this CTA's slice in index order, 1024 tokens at a time, with a block-uniform trip count (the callbacks
    // vote and scan); the first KPT rounds take their keys from registers
    auto for_each_round = [&](auto&& fn) {
#pragma unroll
      for (int it = 0; it < KPT; ++it)
        if (lo + it * NT < hi) { const int i = lo + it * NT + tid; fn(i, i < hi, c_key[it]); }
      for (int c0 = lo + KPT * NT; c0 < hi; c0 += NT) { const int i = c0 + tid; fn(i, i < hi, i < hi ? float_key(mas[i]) : 0u); }
    };
    if (p.select_mode != MAS_SELECT_THRESHOLD) {
      int kk = seg.keep_k < n ? seg.keep_k : n;
      if (p.select_mode == MAS_SELECT_ADAPTIVE) {
        // NEXT-3 (beta_m >= 1 - MAS_m): the smallest retention the constraint admits, from the segment score the
        // fuse launch left in seg_out; the decision is taken in double on the fp32 MAS_s
        const double want = ceil((1.0 - (double)a.seg_out[sidx].mas) * (double)n - 1e-9);
        kk = want < 1.0 ? 1 : (want > (double)n ? n : (int)want);
      }
      const int k_total = kk;
      const bool static_off = p.select_mode == MAS_SELECT_TOPK;   // else positions are data dependent: k_compact_idx writes kept_idx
      unsigned prefix = 0, maskbits = 0;
      if (tid < 256) { sm.hist[0][tid] = 0; sm.hist[1][tid] = 0; sm.hist[2][tid] = 0; sm.hist[3][tid] = 0; }
      __syncthreads();
#pragma unroll 1
      for (int pass = 0; pass < 4; ++pass) {
        const int shift = 24 - 8 * pass;
        for_each_round([&](int, bool valid, unsigned key) {
          const bool act = valid && (key & maskbits) == prefix;
          const unsigned bin = (key >> shift) & 255u;
          if (act) atomicAdd(&sm.hist[pass][bin], 1u);
        });
        __syncthreads();
        const unsigned* hsrc = sm.hist[pass];
        if (nc > 1) {   // cluster-wide histogram: thread b sums bin b over the peers (independent remote loads) into a
          cluster_sync_all();   // private array, so the peers' bins are never overwritten: one cluster barrier per pass
          if (tid < 256) {
            unsigned v[8];
#pragma unroll
            for (unsigned r = 0; r < 8; ++r) v[r] = r < nc ? dsmem_read(&sm.hist[pass][tid], r) : 0u;
            sm.htot[tid] = ((v[0] + v[1]) + (v[2] + v[3])) + ((v[4] + v[5]) + (v[6] + v[7]));
          }
          __syncthreads();
          hsrc = sm.htot;
        }
        if (warp == 0) {   // find the bin where the cumulative count (over the whole cluster) reaches kk
          unsigned loc[8], tot = 0;
#pragma unroll
          for (int b = 0; b < 8; ++b) { loc[b] = hsrc[lane * 8 + b]; tot += loc[b]; }
          unsigned inc = tot;
#pragma unroll
          for (int o = 1; o < 32; o <<= 1) { unsigned u = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += u; }
          unsigned exc = inc - tot;
          const bool mine = exc < (unsigned)kk && (unsigned)kk <= inc;   // exactly one lane
          if (mine) {
            unsigned run = exc;
            int bin = 0;
#pragma unroll
            for (int b = 0; b < 8; ++b) { if (run < (unsigned)kk && (unsigned)kk <= run + loc[b]) { bin = b; break; } run += loc[b]; }
            sm.bcast[0] = lane * 8 + bin;
            sm.bcast[1] = (int)run;   // elements strictly below the chosen bin
          }
        }
        __syncthreads();
        prefix |= (unsigned)sm.bcast[0] << shift;
        maskbits |= 255u << shift;
        kk -= sm.bcast[1];
        __syncthreads();
      }
      // prefix = key of the k-th smallest; keep every key < prefix and the first kk keys == prefix (index order)
      int run_less = 0, run_eq = 0;
      if (nc > 1) {   // kept tokens of the lower-ranked CTAs come first: exchange the per-CTA (less, equal) counts
        int cl = 0, ce = 0;
        for_each_round([&](int, bool valid, unsigned key) { cl += valid && key < prefix; ce += valid && key == prefix; });
        double dl = cl, de = ce, d0 = 0;
        block_sum3(sm, dl, de, d0);
        if (tid == 0) { sm.cx_i[0] = (int)dl; sm.cx_i[1] = (int)de; }
        cluster_sync_all();
        int pl = 0, pe = 0;
        if ((unsigned)lane < rank) { pl = dsmem_read(&sm.cx_i[0], (unsigned)lane); pe = dsmem_read(&sm.cx_i[1], (unsigned)lane); }
        for (int o = 16; o > 0; o >>= 1) { pl += __shfl_xor_sync(0xffffffffu, pl, o); pe += __shfl_xor_sync(0xffffffffu, pe, o); }
        run_less = pl; run_eq = pe;
      }
      const int64_t off = seg.kept_off_static;
      for_each_round([&](int i, bool valid, unsigned key) {
        const int fl = valid && key < prefix, fe = valid && key == prefix;
        int pl, pe, tl, te;
        block_scan2(sm, fl, fe, pl, pe, tl, te);
        const int eq_before = run_eq + pe;
        const bool keep = fl || (fe && eq_before < kk);
        if (valid) {
          if (a.keep_mask) a.keep_mask[base + i] = keep ? 1 : 0;
          if (keep && a.kept_idx && static_off) {
            const int64_t pos = off + run_less + pl + (eq_before < kk ? eq_before : kk);
            if (pos < a.cap_rows) a.kept_idx[pos] = (int32_t)(base + i);
          }
        }
        run_less += tl; run_eq += te;
      });
      if (rank == 0 && tid == 0) {
        a.seg_nkept[sidx] = k_total;
        if (a.seg_out) a.seg_out[sidx].n_kept = k_total;
      }
    } else {
      int cnt = 0;
      const unsigned cut_key = float_key(p.cut);
      for_each_round([&](int i, bool valid, unsigned key) {
        const bool keep = valid && key <= cut_key;     // the key order is the float order (and -0 == +0)
        if (valid && a.keep_mask) a.keep_mask[base + i] = keep ? 1 : 0;
        cnt += keep;
      });
      double dc = cnt, d1 = 0, d2 = 0;
      cluster_sum3(sm, 3, nc, dc, d1, d2);
      if (rank == 0 && tid == 0) {
        a.seg_nkept[sidx] = (int)dc;
        if (a.seg_out) a.seg_out[sidx].n_kept = (int)dc;
      }
    }
  }

  // ---- last cluster: per-request softmax + Eq. 7, and the kept_off table (rank 0 only)
  if (nc > 1) cluster_sync_all();   // no CTA leaves while a peer may still read its shared memory
  if (rank != 0) return;
  __threadfence();
  __syncthreads();
  if (tid == 0) sm.bcast[2] = (atomicAdd(a.done_counter, 1u) == (unsigned)a.n_segs - 1u) ? 1 : 0;
  __syncthreads();
  if (!sm.bcast[2]) return;
  __threadfence();
  if (FUSE && a.seg_out) {
    volatile mas_segment_out* so = a.seg_out;
    for (int r = tid; r < a.n_requests; r += NT) {
      const int k0 = a.req_seg_off[r], k1 = a.req_seg_off[r + 1];
      float mx = -INFINITY;
      for (int k = k0; k < k1; ++k) mx = fmaxf(mx, p.kappa * so[k].alpha_mean);
      float zsum = 0.f;
      for (int k = k0; k < k1; ++k) zsum += expf(p.kappa * so[k].alpha_mean - mx);
      for (int k = k0; k < k1; ++k) {
        const float beta = expf(p.kappa * so[k].alpha_mean - mx) / zsum;
        const float at = a.segs[k].n_frames > 1 ? p.lambda_temp : 0.f;
        so[k].beta = beta;
        so[k].mas = 1.0f - beta * (1.0f - p.lambda_spatial * so[k].rho_spatial - at * (1.0f - so[k].gamma_avg));
      }
    }
  }
  if (SELECT && a.kept_off) {
    if (p.select_mode == MAS_SELECT_TOPK) {
      for (int k = tid; k < a.n_segs; k += NT) a.kept_off[k] = a.segs[k].kept_off_static;
      if (tid == 0) a.kept_off[a.n_segs] = a.segs[a.n_segs - 1].kept_off_static + a.segs[a.n_segs - 1].keep_k;
    } else {
      volatile int32_t* nk = a.seg_nkept;
      long long run = 0;
      for (int c0 = 0; c0 < a.n_segs; c0 += NT) {
        const int k = c0 + tid;
        const int v = k < a.n_segs ? nk[k] : 0;
        // inclusive scan of v over the block (values up to 2^31 in total fit a long long running sum)
        int inc = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { int u = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += u; }
        __syncthreads();
        if (lane == 31) sm.ired[0][warp] = inc;
        __syncthreads();
        int wv = lane < (NT >> 5) ? sm.ired[0][lane] : 0, winc = wv;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { int u = __shfl_up_sync(0xffffffffu, winc, o); if (lane >= o) winc += u; }
        const int wexc = __shfl_sync(0xffffffffu, winc - wv, warp);
        const int tot = __shfl_sync(0xffffffffu, winc, 31);
        if (k < a.n_segs) a.kept_off[k] = run + wexc + inc - v;
        run += tot;
      }
      if (tid == 0) a.kept_off[a.n_segs] = run;
    }
  }
  if (tid == 0) *a.done_counter = 0u;
}

// Threshold mode only: index compaction once kept_off is known (one CTA per segment, ordered ballot + scan).
__global__ void __launch_bounds__(kSegThreads) k_compact_idx(const DevSeg* segs, const uint8_t* keep_mask, const int64_t* kept_off,
                                                             int32_t* kept_idx, int64_t cap_rows) {
  __shared__ SegSmem sm;
  pdl_launch_dependents();
  pdl_wait();
  const DevSeg seg = segs[blockIdx.x];
  const int64_t off = kept_off[blockIdx.x];
  int run = 0;
  for (int c0 = 0; c0 < seg.n_rows; c0 += kSegThreads) {
    const int i = c0 + threadIdx.x;
    const int f = i < seg.n_rows && keep_mask[seg.row0 + i];
    int pf, pz, tf, tz;
    block_scan2(sm, f, 0, pf, pz, tf, tz);
    if (f) {
      const int64_t pos = off + run + pf;
      if (pos < cap_rows) kept_idx[pos] = (int32_t)(seg.row0 + i);
    }
    run += tf;
  }
}

// K3 (a6): one warp per kept row, 16-byte copies, four in flight per lane.
__global__ void __launch_bounds__(256) k_gather(const char* __restrict__ X, char* __restrict__ Y, const int32_t* __restrict__ kept_idx,
                                                const int64_t* __restrict__ total_ptr, int64_t cap_rows, int row_bytes) {
  const int lane = threadIdx.x & 31;
  pdl_launch_dependents();   // a kernel chained behind the gather (the learned-heads finish) may be scheduled as SMs free up
  pdl_wait();
  const int64_t total = *total_ptr < cap_rows ? *total_ptr : cap_rows;
  const int64_t n_warps = (int64_t)gridDim.x * 8;
  const int n16 = row_bytes >> 4;
  for (int64_t j = (int64_t)blockIdx.x * 8 + (threadIdx.x >> 5); j < total; j += n_warps) {
    const uint4* src = reinterpret_cast<const uint4*>(X + (int64_t)kept_idx[j] * row_bytes);
    uint4* dst = reinterpret_cast<uint4*>(Y + j * row_bytes);
    int i = lane;
    for (; i + 96 < n16; i += 128) {
      uint4 v0 = ld_nc16(src + i), v1 = ld_nc16(src + i + 32), v2 = ld_nc16(src + i + 64), v3 = ld_nc16(src + i + 96);
      st_na16(dst + i, v0); st_na16(dst + i + 32, v1); st_na16(dst + i + 64, v2); st_na16(dst + i + 96, v3);
    }
    for (; i < n16; i += 32) st_na16(dst + i, ld_nc16(src + i));
  }
}

// mas_score on the tcgen05 path: gamma = sqrt(D) / (|x_t| + |x_{t-1}|) from the score kernel's sqrt(D) and s (the same
// arithmetic as k_segment's in-place finish); key-frame rows 1, single-frame segments 0
__global__ void __launch_bounds__(256) k_gamma_finish(const DevSeg* __restrict__ segs, const DevTile* __restrict__ tiles,
                                                      const float* __restrict__ s, float* __restrict__ gamma, float sqrt_d) {
  const DevTile tile = tiles[blockIdx.x];
  const DevSeg seg = segs[tile.seg];
  for (int r = threadIdx.x; r < tile.n_rows; r += blockDim.x) {
    const int64_t row = (int64_t)tile.row_start + r;
    float gi = 0.f;
    if (seg.n_frames > 1) {
      if (row - seg.row0 < seg.n_patches) gi = 1.0f;
      else { const float den = (s[row] + s[row - seg.n_patches]) * sqrt_d; gi = den > 0.f ? gamma[row] / den : 0.f; }
    }
    gamma[row] = gi;
  }
}

// staged mas_spatial second phase: m_spatial from s (per-segment standardise + sigmoid, Eq. 3)
__global__ void __launch_bounds__(kSegThreads) k_spatial_finish(const DevSeg* segs, DevParams p, const float* s, float* m_spatial) {
  __shared__ SegSmem sm;
  const DevSeg seg = segs[blockIdx.x];
  const int n = seg.n_rows;
  const int64_t base = seg.row0;
  double ss = 0, d1 = 0, d2 = 0;
  for (int i = threadIdx.x; i < n; i += kSegThreads) ss += (double)s[base + i];
  block_sum3(sm, ss, d1, d2);
  const double mu = ss / n;
  double vs = 0;
  for (int i = threadIdx.x; i < n; i += kSegThreads) { const double e = (double)s[base + i] - mu; vs += e * e; }
  d1 = d2 = 0;
  block_sum3(sm, vs, d1, d2);
  const double den = fmax(sqrt(vs / n), 1e-6 * mu);
  const float inv = den > 0.0 ? (float)(1.0 / den) : 0.f;
  for (int i = threadIdx.x; i < n; i += kSegThreads)
    m_spatial[base + i] = sigmoidf_acc(p.spatial_gain * ((float)((double)s[base + i] - mu) * inv) + p.spatial_bias);
}

}  // namespace msas
