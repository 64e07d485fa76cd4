// k_entropy.cuh — NEXT-4: draft-confidence entropy of Eq. 9 and the speculate rule of Eq. 10
// (PAPER.md:141-149).  For each decode step (one row of logits over the vocabulary): p = softmax(l),
// H = -sum_v p_v log p_v, Speculate = [H <= theta_conf].  A pure streaming reduction: every logit is read once with
// 16-byte loads; each thread keeps an online (max, sum e^{l-m}, sum (l-m) e^{l-m}) triple in base-2 units, rescaled at most
// once per 16-byte group: FFMA + ex2 + FADD + FFMA per logit.  HBM-bound: V * e bytes per row.
//   k_entropy_partial  grid (splits, rows): CTA (s, r) reduces columns [s * chunk, (s+1) * chunk) of row r to one triple
//   k_entropy_finish   one warp per row merges the `splits` triples: H = log Z - T / Z
#pragma once
#include "msas_internal.cuh"

namespace msas {

// Everything is kept in base-2 units so that one FFMA + one ex2 serve each logit: m = max l * log2(e),
// z = sum 2^{u}, t = sum u 2^{u} with u = l * log2(e) - m  (so e^{l - max} = 2^{u}).
struct EntTriple { float m, z, t; };
constexpr float kLog2e = 1.4426950408889634f, kLn2 = 0.6931471805599453f;

__device__ __forceinline__ float ex2f(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

__device__ __forceinline__ EntTriple ent_merge(const EntTriple& a, const EntTriple& b) {
  if (a.z == 0.f) return b;
  if (b.z == 0.f) return a;
  EntTriple r;
  r.m = fmaxf(a.m, b.m);
  const float da = a.m - r.m, db = b.m - r.m;          // <= 0
  const float ea = ex2f(da), eb = ex2f(db);
  r.z = a.z * ea + b.z * eb;
  r.t = (a.t + da * a.z) * ea + (b.t + db * b.z) * eb;
  return r;
}
// fold one 16-byte group of logits into the running triple: one rescale check, then FFMA + ex2 + FADD + FFMA per logit
template <int N, bool FULL>
__device__ __forceinline__ void ent_fold(EntTriple& acc, const float (&x)[N], int n_valid) {
  float gm = x[0];
#pragma unroll
  for (int k = 1; k < N; ++k) if (FULL || k < n_valid) gm = fmaxf(gm, x[k]);
  gm *= kLog2e;
  if (gm > acc.m) {                                     // new maximum: rescale what has been summed so far
    if (acc.z > 0.f) { const float dm = acc.m - gm, e = ex2f(dm); acc.t = (acc.t + dm * acc.z) * e; acc.z *= e; }
    acc.m = gm;
  }
#pragma unroll
  for (int k = 0; k < N; ++k)
    if (FULL || k < n_valid) {
      // masked logits (-inf, e.g. after top-k filtering) contribute 0 (0 ln 0 = 0): the clamp turns -inf, and the NaN of
      // -inf + inf while nothing finite has been seen yet, into an exponent whose 2^u flushes to exactly 0
      const float u = fmaxf(fmaf(x[k], kLog2e, -acc.m), -200.f), e = ex2f(u);
      acc.z += e; acc.t = fmaf(u, e, acc.t);
    }
}

template <int DT>   // 0: fp32, 1: bf16
__global__ void __launch_bounds__(256) k_entropy_partial(const void* __restrict__ logits, int64_t V, int64_t row_stride, int64_t chunk,
                                                          EntTriple* __restrict__ part) {
  constexpr int EPV = DT == 1 ? 8 : 4;                  // elements per 16-byte vector
  pdl_launch_dependents();                              // the finish kernel may be staged; it waits for this grid
  const int64_t row = blockIdx.y;
  const int64_t c0 = (int64_t)blockIdx.x * chunk, c1 = c0 + chunk < V ? c0 + chunk : V;   // chunk is a multiple of EPV
  const char* base = static_cast<const char*>(logits) + row * row_stride * (DT == 1 ? 2 : 4);
  EntTriple acc{-INFINITY, 0.f, 0.f};
  constexpr int ESZ = DT == 1 ? 2 : 4;
  auto unpack = [](const uint4& v, float (&x)[EPV]) {
    if (DT == 1) {
      const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
      for (int k = 0; k < 4; ++k) { x[(2 * k) % EPV] = bf_lo(w[k]); x[(2 * k + 1) % EPV] = bf_hi(w[k]); }
    } else {
      x[0] = __uint_as_float(v.x); x[1] = __uint_as_float(v.y); x[2 % EPV] = __uint_as_float(v.z); x[3 % EPV] = __uint_as_float(v.w);
    }
  };
  int64_t c = c0 + (int64_t)threadIdx.x * EPV;
  // main loop: four independent 16-byte loads in flight per thread (64 B x 2048 threads = 128 KB per SM), then the arithmetic
  for (; c + 3 * 256 * EPV + EPV <= c1; c += 4 * 256 * EPV) {
    uint4 v[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) v[i] = ld_nc16(base + (c + (int64_t)i * 256 * EPV) * ESZ);
#pragma unroll
    for (int i = 0; i < 4; ++i) { float x[EPV]; unpack(v[i], x); ent_fold<EPV, true>(acc, x, EPV); }
  }
  for (; c < c1; c += 256 * EPV) {
    const int nv = c1 - c < EPV ? (int)(c1 - c) : EPV;
    float x[EPV];
    if (nv == EPV) {
      unpack(ld_nc16(base + c * ESZ), x);
      ent_fold<EPV, true>(acc, x, nv);
    } else {                                            // ragged end of the row: element loads
#pragma unroll
      for (int k = 0; k < EPV; ++k) {
        x[k] = 0.f;
        if (k < nv) x[k] = DT == 1 ? __uint_as_float((uint32_t)reinterpret_cast<const unsigned short*>(base)[c + k] << 16)
                                   : reinterpret_cast<const float*>(base)[c + k];
      }
      ent_fold<EPV, false>(acc, x, nv);
    }
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
  pdl_wait();
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
    const float h = acc.z > 0.f ? kLn2 * (log2f(acc.z) - acc.t / acc.z) : 0.f;   // H = ln Z - E_p[l - max], from base-2 units
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
