// k_score_simple.cuh — first-generation score kernels:
//   k_qprep        a0  qinv_j = 1/||q_j||                                   (S0, prompt embedding of Eq. 6)
//   k_rowstats     a1/a2 staged: one warp per row, s_i and gamma_i          (Eq. 3 statistic PAPER.md:91; Eq. 5)
//   k_score_mma    a1+a2+a3 in ONE pass over X: rows go global -> registers once (16-byte loads), the same registers
//                  feed the fp32 norm / difference accumulators and the mma.sync A fragments of the relevance
//                  contraction X·Q^T (bf16 in, fp32 accumulate; fp32 inputs are split hi+lo into 3 MMAs).
// These are the generic-shape path (any d % 8 == 0, any L <= 128) and the staged entry points; the tcgen05/TMA
// kernel in k_score_tc.cuh is the fast path for d % 64 == 0 bf16.
#pragma once
#include "msas_internal.cuh"

namespace msas {

struct ScoreArgs {
  const void* X;
  const void* Q;
  const float* qinv;
  const DevSeg* segs;
  const DevTile* tiles;
  float* s;        // may be NULL
  float* gamma;    // may be NULL
  float* rel;      // may be NULL
  float* S_opt;    // may be NULL, [N, kMaxL]
  unsigned long long* sig;   // LSH mode (NEXT-1): Q is the hash matrix R[64, d] shared by all rows; bit k of sig[row] = [r_k . x >= 0]
  // learned-heads mode (NEXT-2): Q is the weight matrix W[64, d] shared by all rows (row 0 = Eq. 3's 1x1 conv, rows 1.. = the
  // z-half of Eq. 6's first layer).  Per row: m_spatial = sigmoid(w_0 . x + heads_bias); per tile: heads_part[tile][0] = number of
  // rows with m_spatial < heads_tau, heads_part[tile][c] = sum over the tile's rows of w_c . x (c = 1..63)
  float* heads_part;
  float* heads_m;
  float heads_bias, heads_tau;
  int d;
};

// ------------------------------------------------------------------------------------------------ a0
template <int DT>
__global__ void __launch_bounds__(256) k_qprep(const void* __restrict__ Q, float* __restrict__ qinv, int64_t n_q, int d) {
  const int lane = threadIdx.x & 31;
  const int64_t row = (int64_t)blockIdx.x * 8 + (threadIdx.x >> 5);
  pdl_launch_dependents();   // the score kernel's CTAs may be scheduled; they wait for this grid before touching global memory
  pdl_wait();                // (launched behind the previous call's last kernel: that one may still read what we are about to write)
  if (row >= n_q) return;
  float acc = 0.f;
  if (DT == 1) {
    const uint4* p = reinterpret_cast<const uint4*>(static_cast<const __nv_bfloat16*>(Q) + row * d);
    for (int i = lane; i < d / 8; i += 32) {
      uint4 v = ld_nc16(p + i);
      uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
      for (int k = 0; k < 4; ++k) { float a = bf_lo(w[k]), b = bf_hi(w[k]); acc = fmaf(a, a, acc); acc = fmaf(b, b, acc); }
    }
  } else {
    const uint4* p = reinterpret_cast<const uint4*>(static_cast<const float*>(Q) + row * d);
    for (int i = lane; i < d / 4; i += 32) {
      uint4 v = ld_nc16(p + i);
      float a = __uint_as_float(v.x), b = __uint_as_float(v.y), c = __uint_as_float(v.z), e = __uint_as_float(v.w);
      acc = fmaf(a, a, acc); acc = fmaf(b, b, acc); acc = fmaf(c, c, acc); acc = fmaf(e, e, acc);
    }
  }
  acc = warp_sum(acc);
  if (lane == 0) qinv[row] = acc > 0.f ? 1.0f / sqrtf(acc) : 0.f;
}

// ------------------------------------------------------------------------------------------------ a1 / a2 staged
// One CTA per tile, 8 warps, one warp per row at a time.  Reads the previous-frame row directly (L2).
template <int DT>
__global__ void __launch_bounds__(256) k_rowstats(ScoreArgs a) {
  const DevTile tile = a.tiles[blockIdx.x];
  const DevSeg seg = a.segs[tile.seg];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int d = a.d;
  const int esz = DT == 1 ? 2 : 4;
  const int n16 = d * esz / 16;
  for (int r = warp; r < tile.n_rows; r += 8) {
    const int64_t row = (int64_t)tile.row_start + r;
    const bool temporal = a.gamma != nullptr && seg.n_frames > 1;
    const bool has_prev = temporal && (row - seg.row0) >= seg.n_patches;
    const uint4* px = reinterpret_cast<const uint4*>(static_cast<const char*>(a.X) + row * (int64_t)d * esz);
    const uint4* pp = reinterpret_cast<const uint4*>(static_cast<const char*>(a.X) + (row - seg.n_patches) * (int64_t)d * esz);
    float n2 = 0.f, n2p = 0.f, D = 0.f;
    for (int i = lane; i < n16; i += 32) {
      uint4 v = ld_nc16(px + i);
      uint4 u = has_prev ? ld_nc16(pp + i) : make_uint4(0, 0, 0, 0);
      uint32_t vw[4] = {v.x, v.y, v.z, v.w}, uw[4] = {u.x, u.y, u.z, u.w};
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        if (DT == 1) {
          float x0 = bf_lo(vw[k]), x1 = bf_hi(vw[k]), p0 = bf_lo(uw[k]), p1 = bf_hi(uw[k]);
          n2 = fmaf(x0, x0, n2); n2 = fmaf(x1, x1, n2);
          n2p = fmaf(p0, p0, n2p); n2p = fmaf(p1, p1, n2p);
          float e0 = x0 - p0, e1 = x1 - p1;
          D = fmaf(e0, e0, D); D = fmaf(e1, e1, D);
        } else {
          float x0 = __uint_as_float(vw[k]), p0 = __uint_as_float(uw[k]);
          n2 = fmaf(x0, x0, n2); n2p = fmaf(p0, p0, n2p);
          float e0 = x0 - p0;
          D = fmaf(e0, e0, D);
        }
      }
    }
    n2 = warp_sum(n2); n2p = warp_sum(n2p); D = warp_sum(D);
    if (lane == 0) {
      if (a.s) a.s[row] = sqrtf(n2 / (float)d);
      if (a.gamma) {
        float g = 0.f;
        if (temporal) {
          if (!has_prev) g = 1.0f;
          else { float den = sqrtf(n2) + sqrtf(n2p); g = den > 0.f ? sqrtf(D) / den : 0.f; }
        }
        a.gamma[row] = g;
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------ a1+a2+a3 fused (mma.sync)
__device__ __forceinline__ void mma_bf16_16816(float (&c)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t b0, uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
               : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
               : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}

// K-permutation used by both operands: inside a 32-column group, quad lane c owns columns 8c..8c+7; MMA #1 contracts
// its first four (as k = 2c,2c+1,2c+8,2c+9), MMA #2 the last four.  The contraction is order-free, so any bijection
// shared by A and B is valid; this one lets every thread fetch its A fragment with one 16-byte global load per row.
//
// Q chunk in shared memory: [Lpad][64 cols] bf16, 128 B per row, 16-byte pieces XOR-swizzled by ((row & 1) << 2) so
// that the 8 lanes of a quarter warp (two rows x four pieces) hit 8 distinct bank groups.
__device__ __forceinline__ int q_piece_off(int row, int piece) { return row * 128 + ((piece ^ ((row & 1) << 2)) << 4); }

template <int DT, int NT>
__device__ __forceinline__ void score_tile_mma(const ScoreArgs& a, const DevTile& tile, const DevSeg& seg, unsigned char* smem) {
  constexpr int LP = NT * 8;                       // padded query count
  constexpr int QBUF = LP * 128;                   // bytes of one bf16 Q chunk
  constexpr int NPLANE = DT == 1 ? 1 : 2;          // fp32: hi and lo planes
  constexpr int PIECES = (LP * 8 + 255) / 256;     // 16-byte pieces per thread per chunk
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, g = lane >> 2, c = lane & 3;
  const bool shared_b = a.sig != nullptr || a.heads_part != nullptr;   // one 64-row B operand for every tile
  const int d = a.d, L = shared_b ? 64 : seg.L;
  const int esz = DT == 1 ? 2 : 4;

  const int rl = warp * 16 + g, rh = rl + 8;
  const bool vlo = rl < tile.n_rows, vhi = rh < tile.n_rows;
  const int64_t row_lo = (int64_t)tile.row_start + (vlo ? rl : tile.n_rows - 1);
  const int64_t row_hi = (int64_t)tile.row_start + (vhi ? rh : tile.n_rows - 1);
  const bool temporal = a.gamma != nullptr && seg.n_frames > 1;
  const bool plo = temporal && (row_lo - seg.row0) >= seg.n_patches;
  const bool phi = temporal && (row_hi - seg.row0) >= seg.n_patches;
  const char* Xb = static_cast<const char*>(a.X);
  const char* x_lo = Xb + row_lo * (int64_t)d * esz;
  const char* x_hi = Xb + row_hi * (int64_t)d * esz;
  const char* p_lo = x_lo - (int64_t)seg.n_patches * d * esz;
  const char* p_hi = x_hi - (int64_t)seg.n_patches * d * esz;
  const char* Qb = static_cast<const char*>(a.Q) + (shared_b ? (int64_t)0 : (int64_t)seg.q0 * d * esz);

  float acc[NT][4];
#pragma unroll
  for (int j = 0; j < NT; ++j) { acc[j][0] = acc[j][1] = acc[j][2] = acc[j][3] = 0.f; }
  float n2l = 0.f, n2h = 0.f, npl = 0.f, nph = 0.f, Dl = 0.f, Dh = 0.f;

  // Q staging: piece p of this thread = (row qr, 8-column piece qp) of the chunk
  auto stage_load = [&](int kc, uint4 (&hi)[PIECES], uint4 (&lo)[PIECES]) {
#pragma unroll
    for (int i = 0; i < PIECES; ++i) {
      const int idx = tid + i * 256;
      const int qr = idx >> 3, qp = idx & 7;
      const int col = kc + qp * 8;
      hi[i] = make_uint4(0, 0, 0, 0);
      lo[i] = make_uint4(0, 0, 0, 0);
      if (idx < LP * 8 && qr < L && col < d) {
        if (DT == 1) {
          hi[i] = ld_nc16(Qb + ((int64_t)qr * d + col) * 2);
        } else {
          float f[8];
          uint4 v0 = ld_nc16(Qb + ((int64_t)qr * d + col) * 4);
          uint4 v1 = (col + 4 < d) ? ld_nc16(Qb + ((int64_t)qr * d + col + 4) * 4) : make_uint4(0, 0, 0, 0);
          f[0] = __uint_as_float(v0.x); f[1] = __uint_as_float(v0.y); f[2] = __uint_as_float(v0.z); f[3] = __uint_as_float(v0.w);
          f[4] = __uint_as_float(v1.x); f[5] = __uint_as_float(v1.y); f[6] = __uint_as_float(v1.z); f[7] = __uint_as_float(v1.w);
          uint32_t h[4], l[4];
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            h[k] = pack_bf16x2(f[2 * k], f[2 * k + 1]);
            l[k] = pack_bf16x2(f[2 * k] - bf_lo(h[k]), f[2 * k + 1] - bf_hi(h[k]));
          }
          hi[i] = make_uint4(h[0], h[1], h[2], h[3]);
          lo[i] = make_uint4(l[0], l[1], l[2], l[3]);
        }
      }
    }
  };
  auto stage_store = [&](int buf, const uint4 (&hi)[PIECES], const uint4 (&lo)[PIECES]) {
#pragma unroll
    for (int i = 0; i < PIECES; ++i) {
      const int idx = tid + i * 256;
      if (idx < LP * 8) {
        const int qr = idx >> 3, qp = idx & 7;
        unsigned char* base = smem + buf * (QBUF * NPLANE);
        *reinterpret_cast<uint4*>(base + q_piece_off(qr, qp)) = hi[i];
        if (DT == 0) *reinterpret_cast<uint4*>(base + QBUF + q_piece_off(qr, qp)) = lo[i];
      }
    }
  };

  uint4 qh[PIECES], ql[PIECES];
  stage_load(0, qh, ql);
  stage_store(0, qh, ql);
  __syncthreads();

  int buf = 0;
  for (int kc = 0; kc < d; kc += 64, buf ^= 1) {
    const bool more = kc + 64 < d;
    if (more) stage_load(kc + 64, qh, ql);
    const unsigned char* qs = smem + buf * (QBUF * NPLANE);
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      if (kc + h * 32 >= d) continue;          // warp-uniform: whole 32-column group is past the row end
      const int col = kc + h * 32 + c * 8;     // this thread's 8 columns
      const bool inb = col < d;                // d % 8 == 0 (bf16) / d % 4 == 0 (fp32); out-of-range lanes feed zeros
      uint32_t al[4], ah[4];                   // bf16x2-packed A fragments (hi part for fp32 input)
      uint32_t bl[4], bh[4];                   // fp32 input only: lo parts
      if (DT == 1) {
        const uint4 z4 = make_uint4(0, 0, 0, 0);
        uint4 vl = inb ? ld_nc16(x_lo + (int64_t)col * 2) : z4, vh = inb ? ld_nc16(x_hi + (int64_t)col * 2) : z4;
        uint4 ul = (plo && inb) ? ld_nc16(p_lo + (int64_t)col * 2) : z4;
        uint4 uh = (phi && inb) ? ld_nc16(p_hi + (int64_t)col * 2) : z4;
        al[0] = vl.x; al[1] = vl.y; al[2] = vl.z; al[3] = vl.w;
        ah[0] = vh.x; ah[1] = vh.y; ah[2] = vh.z; ah[3] = vh.w;
        uint32_t pl[4] = {ul.x, ul.y, ul.z, ul.w}, ph[4] = {uh.x, uh.y, uh.z, uh.w};
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          float x0 = bf_lo(al[k]), x1 = bf_hi(al[k]), y0 = bf_lo(ah[k]), y1 = bf_hi(ah[k]);
          n2l = fmaf(x0, x0, n2l); n2l = fmaf(x1, x1, n2l);
          n2h = fmaf(y0, y0, n2h); n2h = fmaf(y1, y1, n2h);
          if (temporal) {
            float p0 = bf_lo(pl[k]), p1 = bf_hi(pl[k]), r0 = bf_lo(ph[k]), r1 = bf_hi(ph[k]);
            npl = fmaf(p0, p0, npl); npl = fmaf(p1, p1, npl);
            nph = fmaf(r0, r0, nph); nph = fmaf(r1, r1, nph);
            float e0 = x0 - p0, e1 = x1 - p1, f0 = y0 - r0, f1 = y1 - r1;
            Dl = fmaf(e0, e0, Dl); Dl = fmaf(e1, e1, Dl);
            Dh = fmaf(f0, f0, Dh); Dh = fmaf(f1, f1, Dh);
          }
        }
      } else {
        float xl[8], xh[8], pl[8], ph[8];
        auto ld8 = [&](const char* base, bool on, float (&o)[8]) {
          uint4 v0 = on ? ld_nc16(base + (int64_t)col * 4) : make_uint4(0, 0, 0, 0);
          uint4 v1 = (on && col + 4 < d) ? ld_nc16(base + (int64_t)(col + 4) * 4) : make_uint4(0, 0, 0, 0);
          o[0] = __uint_as_float(v0.x); o[1] = __uint_as_float(v0.y); o[2] = __uint_as_float(v0.z); o[3] = __uint_as_float(v0.w);
          o[4] = __uint_as_float(v1.x); o[5] = __uint_as_float(v1.y); o[6] = __uint_as_float(v1.z); o[7] = __uint_as_float(v1.w);
        };
        ld8(x_lo, inb, xl); ld8(x_hi, inb, xh); ld8(p_lo, plo && inb, pl); ld8(p_hi, phi && inb, ph);
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          n2l = fmaf(xl[k], xl[k], n2l); n2h = fmaf(xh[k], xh[k], n2h);
          if (temporal) {
            npl = fmaf(pl[k], pl[k], npl); nph = fmaf(ph[k], ph[k], nph);
            float e = xl[k] - pl[k], f = xh[k] - ph[k];
            Dl = fmaf(e, e, Dl); Dh = fmaf(f, f, Dh);
          }
        }
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          al[k] = pack_bf16x2(xl[2 * k], xl[2 * k + 1]);
          bl[k] = pack_bf16x2(xl[2 * k] - bf_lo(al[k]), xl[2 * k + 1] - bf_hi(al[k]));
          ah[k] = pack_bf16x2(xh[2 * k], xh[2 * k + 1]);
          bh[k] = pack_bf16x2(xh[2 * k] - bf_lo(ah[k]), xh[2 * k + 1] - bf_hi(ah[k]));
        }
      }
      if (a.rel != nullptr || a.S_opt != nullptr || shared_b) {
#pragma unroll
        for (int j = 0; j < NT; ++j) {
          const int qr = j * 8 + g;
          const uint4 b = *reinterpret_cast<const uint4*>(qs + q_piece_off(qr, h * 4 + c));
          mma_bf16_16816(acc[j], al[0], ah[0], al[1], ah[1], b.x, b.y);
          mma_bf16_16816(acc[j], al[2], ah[2], al[3], ah[3], b.z, b.w);
          if (DT == 0) {
            const uint4 bq = *reinterpret_cast<const uint4*>(qs + QBUF + q_piece_off(qr, h * 4 + c));   // lo plane of Q
            mma_bf16_16816(acc[j], al[0], ah[0], al[1], ah[1], bq.x, bq.y);
            mma_bf16_16816(acc[j], al[2], ah[2], al[3], ah[3], bq.z, bq.w);
            mma_bf16_16816(acc[j], bl[0], bh[0], bl[1], bh[1], b.x, b.y);
            mma_bf16_16816(acc[j], bl[2], bh[2], bl[3], bh[3], b.z, b.w);
          }
        }
      }
    }
    if (more) stage_store(buf ^ 1, qh, ql);
    __syncthreads();
  }

  // ---- epilogue: quad reductions, per-row finalisation
  n2l = quad_sum(n2l); n2h = quad_sum(n2h);
  npl = quad_sum(npl); nph = quad_sum(nph);
  Dl = quad_sum(Dl); Dh = quad_sum(Dh);
  if (a.sig != nullptr) {   // NEXT-1: pack the 64 hash bits of each row (this thread holds columns 8j + 2c, 8j + 2c + 1)
    unsigned long long bl = 0ull, bh = 0ull;
#pragma unroll
    for (int j = 0; j < NT; ++j) {
      const int c0 = j * 8 + 2 * c;
      if (c0 < 64) {
        bl |= (unsigned long long)(acc[j][0] >= 0.f) << c0 | (unsigned long long)(acc[j][1] >= 0.f) << (c0 + 1);
        bh |= (unsigned long long)(acc[j][2] >= 0.f) << c0 | (unsigned long long)(acc[j][3] >= 0.f) << (c0 + 1);
      }
    }
    bl |= __shfl_xor_sync(0xffffffffu, bl, 1); bl |= __shfl_xor_sync(0xffffffffu, bl, 2);
    bh |= __shfl_xor_sync(0xffffffffu, bh, 1); bh |= __shfl_xor_sync(0xffffffffu, bh, 2);
    if (c == 0) { if (vlo) a.sig[row_lo] = bl; if (vhi) a.sig[row_hi] = bh; }
    return;
  }
  if (a.heads_part != nullptr) {   // NEXT-2: column 0 -> the spatial map, columns 1..63 -> per-tile column sums (fixed order: no atomics)
    float cs[NT][2];
#pragma unroll
    for (int j = 0; j < NT; ++j) {
      cs[j][0] = (vlo ? acc[j][0] : 0.f) + (vhi ? acc[j][2] : 0.f);
      cs[j][1] = (vlo ? acc[j][1] : 0.f) + (vhi ? acc[j][3] : 0.f);
    }
    if (c == 0) {   // this thread holds column 0 of its two rows
      int below = 0;
      if (vlo) { const float M = sigmoidf_acc(acc[0][0] + a.heads_bias); a.heads_m[row_lo] = M; below += M < a.heads_tau; }
      if (vhi) { const float M = sigmoidf_acc(acc[0][2] + a.heads_bias); a.heads_m[row_hi] = M; below += M < a.heads_tau; }
      cs[0][0] = (float)below;
    }
    float* red = reinterpret_cast<float*>(smem);   // the B-operand buffers are free after the last barrier of the K loop
#pragma unroll
    for (int j = 0; j < NT; ++j)
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        float v = cs[j][e];
        v += __shfl_xor_sync(0xffffffffu, v, 4); v += __shfl_xor_sync(0xffffffffu, v, 8); v += __shfl_xor_sync(0xffffffffu, v, 16);
        if (g == 0 && j * 8 + 2 * c + e < 64) red[warp * 64 + j * 8 + 2 * c + e] = v;
      }
    __syncthreads();
    if (tid < 64) {
      float t = 0.f;
#pragma unroll
      for (int w = 0; w < 8; ++w) t += red[w * 64 + tid];
      a.heads_part[(int64_t)blockIdx.x * 64 + tid] = t;
    }
    return;
  }
  float ml = -INFINITY, mh = -INFINITY;
  const float* qinv = a.qinv + seg.q0;
#pragma unroll
  for (int j = 0; j < NT; ++j) {
    const int c0 = j * 8 + 2 * c;
    if (c0 < L) {
      const float w0 = qinv[c0];
      ml = fmaxf(ml, acc[j][0] * w0); mh = fmaxf(mh, acc[j][2] * w0);
      if (a.S_opt) {
        if (vlo) a.S_opt[row_lo * kMaxL + c0] = acc[j][0];
        if (vhi) a.S_opt[row_hi * kMaxL + c0] = acc[j][2];
      }
    }
    if (c0 + 1 < L) {
      const float w1 = qinv[c0 + 1];
      ml = fmaxf(ml, acc[j][1] * w1); mh = fmaxf(mh, acc[j][3] * w1);
      if (a.S_opt) {
        if (vlo) a.S_opt[row_lo * kMaxL + c0 + 1] = acc[j][1];
        if (vhi) a.S_opt[row_hi * kMaxL + c0 + 1] = acc[j][3];
      }
    }
  }
  ml = quad_max(ml); mh = quad_max(mh);
  if (c == 0) {
    auto finish = [&](bool valid, int64_t row, float n2, float n2p, float D, bool hasp, float m) {
      if (!valid) return;
      if (a.s) a.s[row] = sqrtf(n2 / (float)d);
      if (a.gamma) {
        float gm = 0.f;
        if (temporal) {
          if (!hasp) gm = 1.0f;
          else { float den = sqrtf(n2) + sqrtf(n2p); gm = den > 0.f ? sqrtf(D) / den : 0.f; }
        }
        a.gamma[row] = gm;
      }
      if (a.rel) a.rel[row] = n2 > 0.f ? m / sqrtf(n2) : 0.f;
    };
    finish(vlo, row_lo, n2l, npl, Dl, plo, ml);
    finish(vhi, row_hi, n2h, nph, Dh, phi, mh);
  }
}

// One CTA (8 warps x 16 rows) per tile.  NT (8-query MMA tiles) is chosen per request from L.
template <int DT>
__global__ void __launch_bounds__(256) k_score_mma(ScoreArgs a) {
  extern __shared__ __align__(16) unsigned char smem[];
  const DevTile tile = a.tiles[blockIdx.x];
  const DevSeg seg = a.segs[tile.seg];
  if (seg.L <= 16) score_tile_mma<DT, 2>(a, tile, seg, smem);
  else if (seg.L <= 32) score_tile_mma<DT, 4>(a, tile, seg, smem);
  else if (seg.L <= 64) score_tile_mma<DT, 8>(a, tile, seg, smem);
  else score_tile_mma<DT, 16>(a, tile, seg, smem);
}

// NEXT-1: signatures of the literal LSH probe (Eq. 5): the same one-pass tile kernel with the 64 hash
// rows as its B operand.
template <int DT>
__global__ void __launch_bounds__(256) k_lsh_sig(ScoreArgs a) {
  extern __shared__ __align__(16) unsigned char smem[];
  const DevTile tile = a.tiles[blockIdx.x];
  const DevSeg seg = a.segs[tile.seg];
  score_tile_mma<DT, 8>(a, tile, seg, smem);
}
// NEXT-2: projections of every row on the 64 head weight rows (Eq. 3's conv + the z-half of Eq. 6's first layer)
template <int DT>
__global__ void __launch_bounds__(256) k_heads_proj(ScoreArgs a) {
  extern __shared__ __align__(16) unsigned char smem[];
  const DevTile tile = a.tiles[blockIdx.x];
  const DevSeg seg = a.segs[tile.seg];
  score_tile_mma<DT, 8>(a, tile, seg, smem);
}
// gamma_lsh = popcount(sig_t xor sig_{t-1}) / 64 per patch; keyframe 1; single-frame segments 0
__global__ void __launch_bounds__(128) k_lsh_gamma(const DevSeg* segs, const DevTile* tiles, const unsigned long long* sig, float* gamma) {
  const DevTile tile = tiles[blockIdx.x];
  const DevSeg seg = segs[tile.seg];
  for (int r = threadIdx.x; r < tile.n_rows; r += blockDim.x) {
    const int64_t row = (int64_t)tile.row_start + r;
    float g = 0.f;
    if (seg.n_frames > 1) g = (row - seg.row0) < seg.n_patches ? 1.0f : (float)__popcll(sig[row] ^ sig[row - seg.n_patches]) * (1.0f / 64.0f);
    gamma[row] = g;
  }
}

constexpr int score_mma_smem_bytes(int dt) { return 2 * (16 * 8 * 128) * (dt == 1 ? 1 : 2); }

}  // namespace msas
