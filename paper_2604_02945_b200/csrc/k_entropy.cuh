// k_entropy.cuh — NEXT-4: draft-confidence entropy of Eq. 9 and the speculate rule of Eq. 10
// (PAPER.md:141-149).  For each decode step (one row of logits over the vocabulary): p = softmax(l),
// H = -sum_v p_v log p_v, Speculate = [H <= theta_conf].  A pure streaming reduction: every logit is read once with
// 16-byte loads; each thread keeps an online (max, sum e^{l-m}, sum (l-m) e^{l-m}) triple, rescaled once per 16-byte
// group, so the cost is one ex2 per logit.  HBM-bound: V * e bytes per row.
//   k_entropy_partial  grid (splits, rows): CTA (s, r) reduces columns [s * chunk, (s+1) * chunk) of row r to one triple
//   k_entropy_finish   one warp per row merges the `splits` triples: H = log Z - T / Z
#pragma once
#include "msas_internal.cuh"

namespace msas {

struct EntTriple { float m, z, t; };   // running max, sum e^{l-m}, sum (l-m) e^{l-m}

__device__ __forceinline__ EntTriple ent_merge(const EntTriple& a, const EntTriple& b) {
  if (a.z == 0.f) return b;
  if (b.z == 0.f) return a;
  EntTriple r;
  r.m = fmaxf(a.m, b.m);
  const float da = a.m - r.m, db = b.m - r.m;          // <= 0
  const float ea = __expf(da), eb = __expf(db);
  r.z = a.z * ea + b.z * eb;
  r.t = (a.t + da * a.z) * ea + (b.t + db * b.z) * eb;
  return r;
}
// fold up to 8 logits (one 16-byte group) into the running triple: one rescale, then one exp per logit
template <int N>
__device__ __forceinline__ void ent_fold(EntTriple& acc, const float (&x)[N], int n_valid) {
  float gm = -INFINITY;
#pragma unroll
  for (int k = 0; k < N; ++k) if (k < n_valid) gm = fmaxf(gm, x[k]);
  if (gm > acc.m) {                                     // new maximum: rescale what has been summed so far
    if (acc.z > 0.f) { const float dm = acc.m - gm, e = __expf(dm); acc.t = (acc.t + dm * acc.z) * e; acc.z *= e; }
    acc.m = gm;
  }
#pragma unroll
  for (int k = 0; k < N; ++k)
    if (k < n_valid) { const float u = x[k] - acc.m, e = __expf(u); acc.z += e; acc.t = fmaf(u, e, acc.t); }
}

template <int DT>   // 0: fp32, 1: bf16
__global__ void __launch_bounds__(256) k_entropy_partial(const void* __restrict__ logits, int64_t V, int64_t row_stride, int64_t chunk,
                                                          EntTriple* __restrict__ part) {
  constexpr int EPV = DT == 1 ? 8 : 4;                  // elements per 16-byte vector
  const int64_t row = blockIdx.y;
  const int64_t c0 = (int64_t)blockIdx.x * chunk, c1 = c0 + chunk < V ? c0 + chunk : V;   // chunk is a multiple of EPV
  const char* base = static_cast<const char*>(logits) + row * row_stride * (DT == 1 ? 2 : 4);
  EntTriple acc{-INFINITY, 0.f, 0.f};
  for (int64_t c = c0 + (int64_t)threadIdx.x * EPV; c < c1; c += 256 * EPV) {
    const int nv = c1 - c < EPV ? (int)(c1 - c) : EPV;
    float x[EPV];
    if (nv == EPV) {
      const uint4 v = ld_nc16(base + c * (DT == 1 ? 2 : 4));
      if (DT == 1) {
        const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int k = 0; k < 4; ++k) { x[(2 * k) % EPV] = bf_lo(w[k]); x[(2 * k + 1) % EPV] = bf_hi(w[k]); }
      } else {
        x[0] = __uint_as_float(v.x); x[1] = __uint_as_float(v.y); x[2 % EPV] = __uint_as_float(v.z); x[3 % EPV] = __uint_as_float(v.w);
      }
    } else {                                            // ragged end of the row: element loads
#pragma unroll
      for (int k = 0; k < EPV; ++k) {
        x[k] = 0.f;
        if (k < nv) x[k] = DT == 1 ? __uint_as_float((uint32_t)reinterpret_cast<const unsigned short*>(base)[c + k] << 16)
                                   : reinterpret_cast<const float*>(base)[c + k];
      }
    }
    ent_fold<EPV>(acc, x, nv);
  }
  // block reduction in a fixed order: warp shuffles, then the 8 warp results through shared memory
  __shared__ EntTriple sm[8];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    EntTriple b;
    b.m = __shfl_xor_sync(0xffffffffu, acc.m, o); b.z = __shfl_xor_sync(0xffffffffu, acc.z, o); b.t = __shfl_xor_sync(0xffffffffu, acc.t, o);
    acc = ent_merge(acc, b);
  }
  if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = acc;
  __syncthreads();
  if (threadIdx.x == 0) {
    EntTriple r = sm[0];
    for (int w = 1; w < 8; ++w) r = ent_merge(r, sm[w]);
    part[row * gridDim.x + blockIdx.x] = r;
  }
}

__global__ void __launch_bounds__(128) k_entropy_finish(const EntTriple* __restrict__ part, int splits, int64_t n_rows, float theta_conf,
                                                         float* __restrict__ H, uint8_t* __restrict__ speculate) {
  const int lane = threadIdx.x & 31;
  const int64_t row = (int64_t)blockIdx.x * 4 + (threadIdx.x >> 5);
  if (row >= n_rows) return;
  EntTriple acc{-INFINITY, 0.f, 0.f};
  for (int s = lane; s < splits; s += 32) acc = ent_merge(acc, part[row * splits + s]);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    EntTriple b;
    b.m = __shfl_xor_sync(0xffffffffu, acc.m, o); b.z = __shfl_xor_sync(0xffffffffu, acc.z, o); b.t = __shfl_xor_sync(0xffffffffu, acc.t, o);
    acc = ent_merge(acc, b);
  }
  if (lane == 0) {
    const float h = acc.z > 0.f ? logf(acc.z) - acc.t / acc.z : 0.f;   // H = log Z - E_p[l - m]
    if (H) H[row] = h;
    if (speculate) speculate[row] = h <= theta_conf ? 1 : 0;
  }
}

// number of column splits per row: enough CTAs to fill the machine a few times over, chunks of at least 8 K logits
inline int entropy_splits(int64_t n_rows, int64_t V, int sm_count) {
  int64_t want = (4ll * sm_count + n_rows - 1) / (n_rows > 0 ? n_rows : 1);
  const int64_t max_by_len = (V + 8191) / 8192;
  if (want > max_by_len) want = max_by_len;
  if (want < 1) want = 1;
  if (want > 256) want = 256;
  return (int)want;
}

}  // namespace msas
