// selftest.cpp — a small executable around the CPU oracle for the sanitiser run (TEST INFRASTRUCTURE, NOT THE PRODUCT).
// tests/test_oracle_pins.py builds it with -fsanitize=address,undefined and runs it: a handful of the closed-form pins
// of tests/golden/closed_forms.txt (MSAO §4.1) plus a whole forward pass with ragged shapes, so that
// any out-of-bounds access, misaligned load, signed overflow or uninitialised-size bug in oracle/mas_oracle.cpp trips
// the sanitiser.  It includes the oracle's translation unit directly: there is nothing else to link.
#include "mas_oracle.cpp"

#include <cstdio>
#include <cstdlib>

static int g_fail = 0;
#define CHECK(cond)                                                          \
  do {                                                                       \
    if (!(cond)) { std::printf("FAIL %s:%d %s\n", __FILE__, __LINE__, #cond); ++g_fail; } \
  } while (0)

static bool near(double a, double b, double tol = 1e-15) { return std::fabs(a - b) <= tol; }

static uint16_t bf16_bits(float f) {   // round to nearest even; inputs are finite
  uint32_t u;
  std::memcpy(&u, &f, 4);
  u += 0x7FFFu + ((u >> 16) & 1u);
  return static_cast<uint16_t>(u >> 16);
}

int main() {
  mas_ref_params prm;
  mas_ref_params_default(&prm);
  CHECK(mas_ref_keep_count(576, 0.25) == 144 && mas_ref_keep_count(18432, 0.15) == 2765 && mas_ref_keep_count(1500, 0.40) == 600);

  {   // Eq. 3-4: two rows with RMS 1 and 3 -> z = -1, +1 -> sigma(-1), sigma(+1), rho = 1/2; Eq. 7 single image -> 0.3
    mas_ref_segment seg{0, 1, 0, 1, 2, 1, 0};
    const double s[2] = {1.0, 3.0}, gam[2] = {0, 0}, rel[2] = {0, 0};
    double m[2], mas[2];
    mas_ref_segment_out out;
    CHECK(mas_ref_fuse(&seg, 1, &prm, s, gam, rel, m, mas, &out) == 0);
    CHECK(near(m[0], 0.2689414213699951) && near(m[1], 0.7310585786300049));
    CHECK(out.rho_spatial == 0.5 && near(out.mas, 0.3) && out.beta == 1.0);
  }
  {   // S2: opposite rows -> 1, doubled -> 1/3, identical -> 0 exactly, keyframe -> 1 (fp32 input, T = 4, P = 1, d = 3)
    mas_ref_segment seg{0, 2, 0, 4, 1, 1, 0};
    const float X[12] = {1, 2, -2, -1, -2, 2, -2, -4, 4, -2, -4, 4};
    double g[4];
    CHECK(mas_ref_temporal(&seg, 1, 3, 0, X, g) == 0);
    CHECK(g[0] == 1.0 && near(g[1], 1.0) && near(g[2], 1.0 / 3.0) && g[3] == 0.0);
  }
  {   // S3: hand-expanded dot products (closed_forms.txt S_00 .. S_12), bf16 inputs (small integers are exact)
    mas_ref_segment seg{0, 1, 0, 1, 2, 1, 0};
    const float Xf[8] = {1, 2, 3, 4, 0, -1, 2, -3}, Qf[12] = {1, 0, -1, 2, 2, 2, 2, 2, -1, 3, 0, 1};
    uint16_t X[8], Q[12];
    for (int i = 0; i < 8; ++i) X[i] = bf16_bits(Xf[i]);
    for (int i = 0; i < 12; ++i) Q[i] = bf16_bits(Qf[i]);
    const int64_t q_off[2] = {0, 3};
    double rel[2], S[6];
    CHECK(mas_ref_crossmodal(&seg, 1, q_off, 1, 4, 1, X, Q, rel, S, 3) == 0);
    const double want[6] = {6, 20, 9, -8, -4, -6};
    for (int i = 0; i < 6; ++i) CHECK(S[i] == want[i]);
    CHECK(near(rel[0], 20.0 / (std::sqrt(30.0) * 4.0), 1e-14));
  }
  {   // whole pass on ragged shapes (an image, a short-frame segment, a video), top-k then threshold: bounds and counts
    const int64_t d = 24;
    mas_ref_segment segs[3] = {{0, 1, 0, 1, 37, 9, 0}, {0, 3, 37, 11, 1, 4, 0}, {1, 2, 48, 3, 13, 10, 0}};
    const int64_t N = 37 + 11 + 39, q_off[3] = {0, 5, 6};
    std::vector<float> X(static_cast<size_t>(N * d)), Q(static_cast<size_t>(6 * d));
    uint32_t st = 12345u;
    auto rnd = [&]() { st = st * 1664525u + 1013904223u; return static_cast<float>((st >> 8) & 0xFFFF) / 32768.0f - 1.0f; };
    for (float& v : X) v = rnd();
    for (float& v : Q) v = rnd();
    for (int64_t c = 0; c < d; ++c) X[static_cast<size_t>((48 + 13 + 4) * d + c)] = X[static_cast<size_t>((48 + 4) * d + c)];   // a static patch
    std::vector<double> m(static_cast<size_t>(N)), gam(static_cast<size_t>(N)), rel(static_cast<size_t>(N)), mas(static_cast<size_t>(N));
    std::vector<uint8_t> mask(static_cast<size_t>(N));
    std::vector<int32_t> idx(static_cast<size_t>(N));
    std::vector<float> Y(static_cast<size_t>(N * d));
    int64_t off[4];
    mas_ref_segment_out out[3];
    for (int mode = 0; mode < 2; ++mode) {
      prm.select_mode = mode;
      prm.cut = 0.5;
      const int64_t cap = mode == 0 ? 23 : 5;   // the threshold run overflows its cap on purpose
      CHECK(mas_ref_forward(segs, 3, q_off, 2, d, 0, &prm, X.data(), Q.data(), nullptr, m.data(), gam.data(), rel.data(), mas.data(), out,
                            mask.data(), idx.data(), off, Y.data(), cap) == 0);
      CHECK(gam[48 + 13 + 4] == 0.0 && gam[48] == 1.0 && gam[0] == 0.0);
      CHECK(near(out[0].beta + out[1].beta, 1.0, 1e-14) && out[2].beta == 1.0);
      int64_t kept = 0;
      for (int64_t i = 0; i < N; ++i) { CHECK(mas[static_cast<size_t>(i)] >= 0.0 && mas[static_cast<size_t>(i)] <= 1.0); kept += mask[static_cast<size_t>(i)]; }
      CHECK(off[3] == kept);
      if (mode == 0) CHECK(kept == 23 && out[0].n_kept == 9 && out[1].n_kept == 4 && out[2].n_kept == 10);
      for (int64_t j = 0; j < std::min(kept, cap); ++j)
        CHECK(std::memcmp(&Y[static_cast<size_t>(j * d)], &X[static_cast<size_t>(idx[static_cast<size_t>(j)] * d)], static_cast<size_t>(d) * 4) == 0);
    }
  }
  if (g_fail == 0) std::printf("oracle selftest ok\n");
  return g_fail == 0 ? 0 : 1;
}
