// mas_oracle.cpp — the CPU ORACLE of the MAS pass.  TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load this library.
// It shares no code, header, table or helper with the CUDA path (paper_2604_02945_b200/csrc): the structs below are
// re-declared here on purpose.
//
// What it is: the plain definition of SPEC.md S0-S5 (paper: MSAO, arxiv/paper_2604_02945, §4.1, PAPER.md:81-124,
// Eq. 3-7; constants PAPER.md:255), written out step by step, single thread, every sum a `double` accumulated in
// index order, inputs converted exactly (bf16 -> double, fp32 -> double). No blocking, fusion or reordering.
//
// NEXT-4 (mas_ref_draft_entropy): pinned by uniform -> log V, one-hot -> 0, the two-level closed form, shift invariance and
// scipy.stats.entropy of a float64 softmax.
// NEXT-2 (mas_ref_learned_heads): pinned by a hand-worked two-segment example (tests/golden/closed_forms.txt, heads_*), the
// ReLU clip it contains, w_sp = 0 -> M = sigmoid(b_sp), a dead hidden layer -> uniform beta, token-order invariance and
// numpy float64 matrix products.
// NEXT-3 (select_mode 2 of mas_ref_select_compact): pinned by worked counts (MAS_s 0.3, N 10 -> 7; 1 -> 1; 0 -> N) and minimality.
// NEXT-3 (mas_ref_spatial_pool, mas_ref_merge_dropped, mas_ref_gather_residual): pinned by scipy.ndimage.uniform_filter (sum / count),
// k = 1 identity, hand-counted corner / edge / centre windows; numpy masked means, the identity n_dropped * mean + kept sum = frame
// sum; static video -> zero residuals, key frames -> copies, residual + previous = original exactly on small integers.
// NEXT-1 (mas_ref_temporal_lsh): pinned by explicit signs of hand-expanded projections, identical / negated rows,
// power-of-two scaling, and the collision law E[gamma] = theta / pi.
//
// Pins (tests/test_oracle_pins.py, `-m "not gpu"`): explicit hand-expanded dot products, closed forms
// (sigma(+-1), 1/sqrt2, 1/3, sin(theta/2)), invariances (query permutation, power-of-two scaling, duplicate query),
// softmax identities, Eq. 7 special cases, brute-force sort/count for selection, numpy float64 cross-checks,
// AR(1) statistical law.  Free conventions shared by both sides and therefore not pinnable by mathematics:
// kappa = 10 (G20) and the standardisation floors 1e-6 (G18).
//
// Build: g++ -O2 -shared -fPIC (no -ffast-math, no OpenMP): oracle/mas_ref.py build().  oracle/selftest.cpp runs a few of the
// pins and a ragged whole pass under -fsanitize=address,undefined (tests/test_oracle_pins.py).

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

extern "C" {

typedef struct {
  int32_t request;
  int32_t modality;
  int64_t row0;
  int32_t n_frames;   // T
  int32_t n_patches;  // P
  int32_t keep_k;
  int32_t reserved_;
} mas_ref_segment;

typedef struct {
  double lambda_spatial, lambda_temp, tau_s, kappa;
  double spatial_gain, spatial_bias, rel_gain, rel_bias;
  double cut;
  int32_t select_mode;  // 0 = top-k, 1 = threshold
  int32_t pad_;
} mas_ref_params;

typedef struct {
  double rho_spatial, gamma_avg, alpha_mean, beta, mas, mean_s, std_s, mean_r, std_r;
  int64_t n_tokens, n_kept;
} mas_ref_segment_out;

enum { REF_F32 = 0, REF_BF16 = 1 };

}  // extern "C"

namespace {

// exact element -> double
inline double elem(const void* base, int dtype, int64_t idx) {
  if (dtype == REF_BF16) {
    uint16_t h = static_cast<const uint16_t*>(base)[idx];
    uint32_t u = static_cast<uint32_t>(h) << 16;
    float f;
    std::memcpy(&f, &u, 4);
    return static_cast<double>(f);
  }
  return static_cast<double>(static_cast<const float*>(base)[idx]);
}

inline int64_t elem_bytes(int dtype) { return dtype == REF_BF16 ? 2 : 4; }

inline double sigmoid(double u) { return 1.0 / (1.0 + std::exp(-u)); }

// S0: n2_i = sum_c x_ic^2
double row_n2(const void* X, int dtype, int64_t row, int64_t d) {
  double acc = 0.0;
  for (int64_t c = 0; c < d; ++c) {
    double v = elem(X, dtype, row * d + c);
    acc += v * v;
  }
  return acc;
}

}  // namespace

extern "C" {

void mas_ref_params_default(mas_ref_params* p) {
  p->lambda_spatial = 0.6;
  p->lambda_temp = 0.4;
  p->tau_s = 0.3;
  p->kappa = 10.0;          // SPEC G20
  p->spatial_gain = 1.0;
  p->spatial_bias = 0.0;
  p->rel_gain = 1.0;
  p->rel_bias = 0.0;
  p->cut = 0.5;
  p->select_mode = 0;
  p->pad_ = 0;
}

// SPEC S5 / G16
int32_t mas_ref_keep_count(int64_t n, double ratio) {
  double c = std::ceil(ratio * static_cast<double>(n) - 1e-9);
  int64_t k = static_cast<int64_t>(c);
  if (k < 1) k = 1;
  if (k > n) k = n;
  return static_cast<int32_t>(k);
}

// S1 first half (Eq. 3's pooled statistic, G1): s_i = sqrt(n2_i / d) for every row of every segment.
int mas_ref_rms(const mas_ref_segment* segs, int32_t n_segs, int64_t d, int dtype, const void* X, double* s) {
  for (int32_t k = 0; k < n_segs; ++k) {
    int64_t n = static_cast<int64_t>(segs[k].n_frames) * segs[k].n_patches;
    for (int64_t i = segs[k].row0; i < segs[k].row0 + n; ++i) s[i] = std::sqrt(row_n2(X, dtype, i, d) / static_cast<double>(d));
  }
  return 0;
}

// S2 (Eq. 5 in exact form; G4-G6): per-patch relative L2 change against the previous frame.
int mas_ref_temporal(const mas_ref_segment* segs, int32_t n_segs, int64_t d, int dtype, const void* X, double* gamma) {
  for (int32_t k = 0; k < n_segs; ++k) {
    const int64_t T = segs[k].n_frames, P = segs[k].n_patches, r0 = segs[k].row0;
    for (int64_t t = 0; t < T; ++t) {
      for (int64_t p = 0; p < P; ++p) {
        const int64_t i = r0 + t * P + p;
        if (T == 1) { gamma[i] = 0.0; continue; }   // temporal term not applicable
        if (t == 0) { gamma[i] = 1.0; continue; }   // keyframe rule G6
        const int64_t j = i - P;                    // same patch, previous frame
        double D = 0.0;
        for (int64_t c = 0; c < d; ++c) {
          double diff = elem(X, dtype, i * d + c) - elem(X, dtype, j * d + c);
          D += diff * diff;
        }
        double den = std::sqrt(row_n2(X, dtype, i, d)) + std::sqrt(row_n2(X, dtype, j, d));
        gamma[i] = den > 0.0 ? std::sqrt(D) / den : 0.0;
      }
    }
  }
  return 0;
}

// NEXT-1: the LITERAL probe of Eq. 5: K = 64 sign-random-projection hashes
// h_k(x) = [r_k . x >= 0] from a supplied matrix R[64, d]; sim = (1/K) sum_k 1[h_k(f_t) = h_k(f_{t-1})],
// gamma = 1 - sim = popcount(sig_t xor sig_{t-1}) / 64.  Per patch (G5), keyframe gamma = 1 (G6), T = 1 -> 0.
// sig[i] bit k = h_k(x_i).  proj_opt (may be NULL): the 64 projections of every row, row-major [N, 64].
int mas_ref_temporal_lsh(const mas_ref_segment* segs, int32_t n_segs, int64_t d, int dtype, const void* X, const void* R,
                         uint64_t* sig, double* proj_opt, double* gamma) {
  for (int32_t k = 0; k < n_segs; ++k) {
    const int64_t T = segs[k].n_frames, P = segs[k].n_patches, r0 = segs[k].row0;
    for (int64_t i = r0; i < r0 + T * P; ++i) {
      uint64_t bits = 0;
      for (int h = 0; h < 64; ++h) {
        double acc = 0.0;
        for (int64_t c = 0; c < d; ++c) acc += elem(R, dtype, (int64_t)h * d + c) * elem(X, dtype, i * d + c);
        if (proj_opt) proj_opt[i * 64 + h] = acc;
        if (acc >= 0.0) bits |= (uint64_t)1 << h;
      }
      sig[i] = bits;
    }
    for (int64_t t = 0; t < T; ++t)
      for (int64_t p = 0; p < P; ++p) {
        const int64_t i = r0 + t * P + p;
        if (T == 1) { gamma[i] = 0.0; continue; }
        if (t == 0) { gamma[i] = 1.0; continue; }
        uint64_t x = sig[i] ^ sig[i - P];
        int cnt = 0;
        while (x) { cnt += (int)(x & 1); x >>= 1; }
        gamma[i] = (double)cnt / 64.0;
      }
  }
  return 0;
}

// NEXT-4: draft-confidence entropy, Eq. 9-10: for each decode step (row) with
// logits l_v over the vocabulary, p = softmax(l), H = - sum_v p_v log p_v (natural log), Speculate = [H <= theta_conf].
// Written as the definition: two passes per row in double (max, then the sums), no online rescaling.
int mas_ref_draft_entropy(const void* logits, int64_t n_rows, int64_t V, int64_t row_stride, int dtype, double theta_conf,
                          double* H, uint8_t* speculate) {
  for (int64_t r = 0; r < n_rows; ++r) {
    double m = -INFINITY;
    for (int64_t v = 0; v < V; ++v) m = std::max(m, elem(logits, dtype, r * row_stride + v));
    double Z = 0.0;
    for (int64_t v = 0; v < V; ++v) Z += std::exp(elem(logits, dtype, r * row_stride + v) - m);
    double h = 0.0;
    for (int64_t v = 0; v < V; ++v) {
      const double lp = elem(logits, dtype, r * row_stride + v) - m - std::log(Z);   // log p_v
      const double pv = std::exp(lp);
      if (pv > 0.0) h -= pv * lp;                                                    // 0 log 0 = 0
    }
    H[r] = h;
    if (speculate) speculate[r] = h <= theta_conf ? 1 : 0;
  }
  return 0;
}

// S3 (Eq. 6, training-free form G9): S_ij = x_i . q_j ; c_ij = S_ij / (|x_i||q_j|) ; r_i = max_j c_ij.
// S_opt (may be NULL): raw dot products, row-major [N, S_stride], columns >= L_r untouched.
int mas_ref_crossmodal(const mas_ref_segment* segs, int32_t n_segs, const int64_t* q_off, int32_t n_requests,
                       int64_t d, int dtype, const void* X, const void* Q, double* rel, double* S_opt, int64_t S_stride) {
  for (int32_t k = 0; k < n_segs; ++k) {
    const int32_t r = segs[k].request;
    if (r < 0 || r >= n_requests) return 1;
    const int64_t q0 = q_off[r], q1 = q_off[r + 1];
    const int64_t n = static_cast<int64_t>(segs[k].n_frames) * segs[k].n_patches;
    std::vector<double> qn(static_cast<size_t>(q1 - q0));
    for (int64_t j = q0; j < q1; ++j) qn[static_cast<size_t>(j - q0)] = std::sqrt(row_n2(Q, dtype, j, d));
    for (int64_t i = segs[k].row0; i < segs[k].row0 + n; ++i) {
      const double xn = std::sqrt(row_n2(X, dtype, i, d));
      double best = 0.0;
      bool first = true;
      for (int64_t j = q0; j < q1; ++j) {
        double S = 0.0;
        for (int64_t c = 0; c < d; ++c) S += elem(X, dtype, i * d + c) * elem(Q, dtype, j * d + c);
        if (S_opt) S_opt[i * S_stride + (j - q0)] = S;
        const double qnj = qn[static_cast<size_t>(j - q0)];
        const double cosv = (xn > 0.0 && qnj > 0.0) ? S / (xn * qnj) : 0.0;
        if (first || cosv > best) { best = cosv; first = false; }
      }
      rel[i] = best;
    }
  }
  return 0;
}

// S1 statistics + S3 statistics + S4 (Eq. 3, 4, 6-softmax, 7).
int mas_ref_fuse(const mas_ref_segment* segs, int32_t n_segs, const mas_ref_params* prm,
                 const double* s, const double* gamma, const double* rel,
                 double* m_spatial, double* mas_tok, mas_ref_segment_out* out) {
  for (int32_t k = 0; k < n_segs; ++k) {
    const int64_t T = segs[k].n_frames, P = segs[k].n_patches, r0 = segs[k].row0, n = T * P;
    const double a = T > 1 ? 1.0 : 0.0;  // temporal applicability
    // S1: population mean / std of s
    double mu_s = 0.0;
    for (int64_t i = r0; i < r0 + n; ++i) mu_s += s[i];
    mu_s /= static_cast<double>(n);
    double var_s = 0.0;
    for (int64_t i = r0; i < r0 + n; ++i) var_s += (s[i] - mu_s) * (s[i] - mu_s);
    const double sd_s = std::sqrt(var_s / static_cast<double>(n));
    const double den_s = std::max(sd_s, 1e-6 * mu_s);
    // S3: population mean / std of rel
    double mu_r = 0.0;
    for (int64_t i = r0; i < r0 + n; ++i) mu_r += rel[i];
    mu_r /= static_cast<double>(n);
    double var_r = 0.0;
    for (int64_t i = r0; i < r0 + n; ++i) var_r += (rel[i] - mu_r) * (rel[i] - mu_r);
    const double sd_r = std::sqrt(var_r / static_cast<double>(n));
    const double den_r = std::max(sd_r, 1e-6);
    int64_t below = 0;
    for (int64_t i = r0; i < r0 + n; ++i) {
      const double z = den_s > 0.0 ? (s[i] - mu_s) / den_s : 0.0;
      const double M = sigmoid(prm->spatial_gain * z + prm->spatial_bias);          // Eq. 3
      if (M < prm->tau_s) ++below;                                                   // Eq. 4, strict <
      const double g = sigmoid(prm->rel_gain * (rel[i] - mu_r) / den_r + prm->rel_bias);
      const double mas = 1.0 - g * (1.0 - prm->lambda_spatial * (1.0 - M) - a * prm->lambda_temp * (1.0 - gamma[i]));  // S4 per token
      if (m_spatial) m_spatial[i] = M;
      mas_tok[i] = mas;
    }
    // S2 aggregate: gamma_avg = mean over t = 1..T-1 of the per-frame patch means
    double gavg = 0.0;
    if (T > 1) {
      for (int64_t t = 1; t < T; ++t) {
        double gt = 0.0;
        for (int64_t p = 0; p < P; ++p) gt += gamma[r0 + t * P + p];
        gavg += gt / static_cast<double>(P);
      }
      gavg /= static_cast<double>(T - 1);
    }
    out[k].rho_spatial = static_cast<double>(below) / static_cast<double>(n);
    out[k].gamma_avg = gavg;
    out[k].alpha_mean = mu_r;
    out[k].mean_s = mu_s;
    out[k].std_s = sd_s;
    out[k].mean_r = mu_r;
    out[k].std_r = sd_r;
    out[k].n_tokens = n;
    out[k].n_kept = 0;
    out[k].beta = 0.0;
    out[k].mas = 0.0;
  }
  // softmax over the segments of each request, then Eq. 7 per segment
  int32_t k0 = 0;
  while (k0 < n_segs) {
    int32_t k1 = k0;
    while (k1 < n_segs && segs[k1].request == segs[k0].request) ++k1;
    double mx = prm->kappa * out[k0].alpha_mean;
    for (int32_t k = k0; k < k1; ++k) mx = std::max(mx, prm->kappa * out[k].alpha_mean);
    double z = 0.0;
    for (int32_t k = k0; k < k1; ++k) z += std::exp(prm->kappa * out[k].alpha_mean - mx);
    for (int32_t k = k0; k < k1; ++k) {
      const double a = segs[k].n_frames > 1 ? 1.0 : 0.0;
      out[k].beta = std::exp(prm->kappa * out[k].alpha_mean - mx) / z;
      out[k].mas = 1.0 - out[k].beta * (1.0 - prm->lambda_spatial * out[k].rho_spatial - a * prm->lambda_temp * (1.0 - out[k].gamma_avg));  // Eq. 7, G8
    }
    k0 = k1;
  }
  return 0;
}

// S5: selection + compaction.  Y may be NULL.  Nothing is written past cap_rows;
// kept_off[n_segs] is always the true total.
int mas_ref_select_compact(const mas_ref_segment* segs, int32_t n_segs, int64_t d, int dtype, const mas_ref_params* prm,
                           const void* X, const double* mas_tok, uint8_t* keep_mask, int32_t* kept_idx, int64_t* kept_off,
                           void* Y, int64_t cap_rows, mas_ref_segment_out* out) {
  int64_t total = 0;
  for (int32_t k = 0; k < n_segs; ++k) {
    const int64_t r0 = segs[k].row0, n = static_cast<int64_t>(segs[k].n_frames) * segs[k].n_patches;
    for (int64_t i = r0; i < r0 + n; ++i) keep_mask[i] = 0;
    if (prm->select_mode == 0 || prm->select_mode == 2) {
      // the keep_k smallest under the strict total order (MAS_i, i): stable sort by value keeps lower index first
      std::vector<int64_t> order(static_cast<size_t>(n));
      for (int64_t i = 0; i < n; ++i) order[static_cast<size_t>(i)] = r0 + i;
      std::stable_sort(order.begin(), order.end(), [&](int64_t a, int64_t b) { return mas_tok[a] < mas_tok[b]; });
      int64_t kk = segs[k].keep_k;
      if (prm->select_mode == 2) {
        // NEXT-3 (adaptive retention): the scheduler's constraint beta_m >= 1 - MAS_m (Eq. 11) read as the
        // smallest admissible retention: keep_k = ceil((1 - MAS_s) N_s), clamped to [1, N_s]; MAS_s from the fuse step
        if (!out) return 1;
        kk = static_cast<int64_t>(std::ceil((1.0 - static_cast<double>(out[k].mas)) * static_cast<double>(n) - 1e-9));
        kk = std::min<int64_t>(n, std::max<int64_t>(1, kk));
      }
      if (kk < 0 || kk > n) return 1;
      for (int64_t j = 0; j < kk; ++j) keep_mask[order[static_cast<size_t>(j)]] = 1;
    } else {
      for (int64_t i = r0; i < r0 + n; ++i) keep_mask[i] = mas_tok[i] <= prm->cut ? 1 : 0;   // G17
    }
    kept_off[k] = total;
    for (int64_t i = r0; i < r0 + n; ++i) {
      if (!keep_mask[i]) continue;
      if (total < cap_rows) {
        if (kept_idx) kept_idx[total] = static_cast<int32_t>(i);
        if (Y) std::memcpy(static_cast<char*>(Y) + total * d * elem_bytes(dtype),
                           static_cast<const char*>(X) + i * d * elem_bytes(dtype), static_cast<size_t>(d * elem_bytes(dtype)));
      }
      ++total;
    }
    if (out) out[k].n_kept = total - kept_off[k];
  }
  kept_off[n_segs] = total;
  return 0;
}

// Whole pass = the staged definitions in order.  Any of m_spatial/gamma/rel may be NULL (scratch is used).
int mas_ref_forward(const mas_ref_segment* segs, int32_t n_segs, const int64_t* q_off, int32_t n_requests,
                    int64_t d, int dtype, const mas_ref_params* prm, const void* X, const void* Q,
                    double* s, double* m_spatial, double* gamma, double* rel, double* mas_tok, mas_ref_segment_out* out,
                    uint8_t* keep_mask, int32_t* kept_idx, int64_t* kept_off, void* Y, int64_t cap_rows) {
  if (n_segs <= 0) { if (kept_off) kept_off[0] = 0; return 0; }
  const int64_t N = segs[n_segs - 1].row0 + static_cast<int64_t>(segs[n_segs - 1].n_frames) * segs[n_segs - 1].n_patches;
  std::vector<double> s_buf, g_buf, r_buf;
  if (!s) { s_buf.resize(static_cast<size_t>(N)); s = s_buf.data(); }
  if (!gamma) { g_buf.resize(static_cast<size_t>(N)); gamma = g_buf.data(); }
  if (!rel) { r_buf.resize(static_cast<size_t>(N)); rel = r_buf.data(); }
  int rc;
  if ((rc = mas_ref_rms(segs, n_segs, d, dtype, X, s))) return rc;
  if ((rc = mas_ref_temporal(segs, n_segs, d, dtype, X, gamma))) return rc;
  if ((rc = mas_ref_crossmodal(segs, n_segs, q_off, n_requests, d, dtype, X, Q, rel, nullptr, 0))) return rc;
  if ((rc = mas_ref_fuse(segs, n_segs, prm, s, gamma, rel, m_spatial, mas_tok, out))) return rc;
  if (keep_mask && kept_off)
    if ((rc = mas_ref_select_compact(segs, n_segs, d, dtype, prm, X, mas_tok, keep_mask, kept_idx, kept_off, Y, cap_rows, out))) return rc;
  return 0;
}

// NEXT-2: the paper's LEARNED heads, with weights supplied by the caller (the trained ones are unpublished).
//   Eq. 3: M_i = sigmoid(w_sp . x_i + b_sp)  -- a 1x1 convolution C -> 1 on each patch's channel vector;
//   Eq. 4:    rho = |{i : M_i < tau_s}| / N_s;
//   Eq. 6: alpha_s = MLP([p ; z_s]) with p = mean of the request's query rows, z_s = mean of the segment's
//     token rows, MLP = one hidden ReLU layer of `hidden` units: alpha = w2 . relu(W1z z + W1p p + b1) + b2 (reading N2);
//   beta = softmax of alpha over the request's segments, as printed (no temperature); Eq. 7 with reading G8.
// W[64, d]: row 0 = w_sp, rows 1..hidden = W1z.  Wp[64, d]: rows 1..hidden = W1p.  b1, w2: entries 1..hidden.  Other rows
// and entries are ignored.  gamma[N] is the temporal probe's output (S2); it is read for segments with T > 1 only.
int mas_ref_learned_heads(const mas_ref_segment* segs, int32_t n_segs, const int64_t* q_off, int64_t d, int dtype,
                          const mas_ref_params* prm, const void* X, const void* Q, const double* gamma, const void* W,
                          const void* Wp, const double* b1, const double* w2, double b_sp, double b2, int32_t hidden,
                          double* m_spatial, mas_ref_segment_out* out) {
  if (hidden < 1 || hidden > 63) return 1;
  std::vector<double> z(static_cast<size_t>(d)), pm(static_cast<size_t>(d));
  for (int32_t k = 0; k < n_segs; ++k) {
    const int64_t T = segs[k].n_frames, P = segs[k].n_patches, r0 = segs[k].row0, n = T * P;
    const int64_t qa = q_off[segs[k].request], qb = q_off[segs[k].request + 1];
    if (qb <= qa) return 1;
    int64_t below = 0;
    for (int64_t i = r0; i < r0 + n; ++i) {
      double u = 0.0;
      for (int64_t c = 0; c < d; ++c) u += elem(W, dtype, c) * elem(X, dtype, i * d + c);
      const double M = sigmoid(u + b_sp);                       // Eq. 3
      if (M < prm->tau_s) ++below;                              // Eq. 4, strict <
      if (m_spatial) m_spatial[i] = M;
    }
    for (int64_t c = 0; c < d; ++c) {                           // z_s, p: plain column means
      double a = 0.0;
      for (int64_t i = r0; i < r0 + n; ++i) a += elem(X, dtype, i * d + c);
      z[static_cast<size_t>(c)] = a / static_cast<double>(n);
      double b = 0.0;
      for (int64_t j = qa; j < qb; ++j) b += elem(Q, dtype, j * d + c);
      pm[static_cast<size_t>(c)] = b / static_cast<double>(qb - qa);
    }
    double alpha = b2;
    for (int32_t h = 1; h <= hidden; ++h) {
      double pre = b1[h];
      for (int64_t c = 0; c < d; ++c) pre += elem(W, dtype, h * d + c) * z[static_cast<size_t>(c)] + elem(Wp, dtype, h * d + c) * pm[static_cast<size_t>(c)];
      alpha += w2[h] * std::max(pre, 0.0);
    }
    double gavg = 0.0;
    if (T > 1) {
      for (int64_t t = 1; t < T; ++t) {
        double gt = 0.0;
        for (int64_t q = 0; q < P; ++q) gt += gamma[r0 + t * P + q];
        gavg += gt / static_cast<double>(P);
      }
      gavg /= static_cast<double>(T - 1);
    }
    out[k].rho_spatial = static_cast<double>(below) / static_cast<double>(n);
    out[k].gamma_avg = gavg;
    out[k].alpha_mean = alpha;
    out[k].mean_s = 0.0; out[k].std_s = 0.0; out[k].mean_r = 0.0; out[k].std_r = 0.0;
    out[k].n_tokens = n; out[k].n_kept = 0; out[k].beta = 0.0; out[k].mas = 0.0;
  }
  int32_t k0 = 0;
  while (k0 < n_segs) {
    int32_t k1 = k0;
    while (k1 < n_segs && segs[k1].request == segs[k0].request) ++k1;
    double mx = out[k0].alpha_mean;
    for (int32_t k = k0; k < k1; ++k) mx = std::max(mx, out[k].alpha_mean);
    double zs = 0.0;
    for (int32_t k = k0; k < k1; ++k) zs += std::exp(out[k].alpha_mean - mx);
    for (int32_t k = k0; k < k1; ++k) {
      const double a = segs[k].n_frames > 1 ? 1.0 : 0.0;
      out[k].beta = std::exp(out[k].alpha_mean - mx) / zs;
      out[k].mas = 1.0 - out[k].beta * (1.0 - prm->lambda_spatial * out[k].rho_spatial - a * prm->lambda_temp * (1.0 - out[k].gamma_avg));  // Eq. 7, G8
    }
    k0 = k1;
  }
  return 0;
}

// NEXT-3, the rest of PAPER.md:98 / 105 ("coarsely compressed", "represented using only the residual difference").
//
// (a) Spatial pooling of the per-token scalar map (Eq. 3's AvgPool, reading G1: a k x k window on the H x W patch grid of every
//     frame, H = P / W; the mean runs over the window cells that lie inside the grid).  Window of cell (i, j): rows
//     i - (k-1)/2 .. i + k/2, columns j - (k-1)/2 .. j + k/2.
int mas_ref_spatial_pool(const mas_ref_segment* segs, int32_t n_segs, const int32_t* grid_w, int32_t k, const double* s, double* out) {
  if (k < 1) return 1;
  for (int32_t q = 0; q < n_segs; ++q) {
    const int64_t T = segs[q].n_frames, P = segs[q].n_patches, r0 = segs[q].row0, W = grid_w[q];
    if (W < 1 || P % W != 0) return 1;
    const int64_t H = P / W, lo = (k - 1) / 2, hi = k / 2;
    for (int64_t t = 0; t < T; ++t)
      for (int64_t i = 0; i < H; ++i)
        for (int64_t j = 0; j < W; ++j) {
          double acc = 0.0;
          int64_t cnt = 0;
          for (int64_t a = i - lo; a <= i + hi; ++a)
            for (int64_t b = j - lo; b <= j + hi; ++b)
              if (a >= 0 && a < H && b >= 0 && b < W) { acc += s[r0 + t * P + a * W + b]; ++cnt; }
          out[r0 + t * P + i * W + j] = acc / static_cast<double>(cnt);
        }
  }
  return 0;
}

// (b) Coarse compression: the dropped tokens (keep_mask = 0) of every frame merged into ONE mean token.  Frames are numbered
//     segment by segment; Ymerge[f] = mean of the frame's dropped rows (zeros when none is dropped), n_dropped[f] their number.
int mas_ref_merge_dropped(const mas_ref_segment* segs, int32_t n_segs, int64_t d, int dtype, const void* X, const uint8_t* keep_mask,
                          double* Ymerge, int64_t* n_dropped) {
  int64_t f = 0;
  for (int32_t q = 0; q < n_segs; ++q)
    for (int64_t t = 0; t < segs[q].n_frames; ++t, ++f) {
      const int64_t P = segs[q].n_patches, r0 = segs[q].row0 + t * P;
      int64_t cnt = 0;
      for (int64_t i = 0; i < P; ++i) cnt += keep_mask[r0 + i] ? 0 : 1;
      n_dropped[f] = cnt;
      for (int64_t c = 0; c < d; ++c) {
        double acc = 0.0;
        for (int64_t i = 0; i < P; ++i)
          if (!keep_mask[r0 + i]) acc += elem(X, dtype, (r0 + i) * d + c);
        Ymerge[f * d + c] = cnt ? acc / static_cast<double>(cnt) : 0.0;
      }
    }
  return 0;
}

// (c) Residual coding of the kept rows: a kept token of frame t >= 1 of a temporal segment is emitted as x_t - x_{t-1} (same
//     patch, previous frame), everything else as a copy.  The difference of two bf16 values is exact in fp32, so the emitted
//     bf16 is its round-to-nearest-even; fp32 inputs: one fp32 subtraction.  Y has the dtype of X.
int mas_ref_gather_residual(const mas_ref_segment* segs, int32_t n_segs, int64_t d, int dtype, const void* X, const int32_t* kept_idx,
                            int64_t n_kept, void* Y) {
  for (int64_t j = 0; j < n_kept; ++j) {
    const int64_t row = kept_idx[j];
    int32_t q = 0;
    while (q + 1 < n_segs && segs[q + 1].row0 <= row) ++q;
    const int64_t P = segs[q].n_patches;
    const bool res = segs[q].n_frames > 1 && row - segs[q].row0 >= P;
    for (int64_t c = 0; c < d; ++c) {
      if (dtype == REF_BF16) {
        float v = static_cast<float>(elem(X, dtype, row * d + c));
        if (res) v -= static_cast<float>(elem(X, dtype, (row - P) * d + c));   // exact
        uint32_t u;
        std::memcpy(&u, &v, 4);
        const uint32_t rnd = ((u >> 16) & 1u) + 0x7FFFu;                         // round to nearest even (finite inputs)
        static_cast<uint16_t*>(Y)[j * d + c] = static_cast<uint16_t>((u + rnd) >> 16);
      } else {
        float v = static_cast<const float*>(X)[row * d + c];
        if (res) v = v - static_cast<const float*>(X)[(row - P) * d + c];
        static_cast<float*>(Y)[j * d + c] = v;
      }
    }
  }
  return 0;
}

}  // extern "C"
