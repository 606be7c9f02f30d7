// ---------------------------------------------------------------------------
// CPU ORACLE for the LPF hot path  --  TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// A plain, slow, single-threaded float64 restatement of what the path computes,
// written from the paper (Ruhe et al., arXiv 2103.15418; /root/reference/PAPER.md)
// and from the readings listed in DESIGN.md ("Readings", R1..R26).  It shares no
// code with the CUDA path (paper_2103_15418_b200/csrc) and neither includes the
// other.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
// --impl reference legs may load this library.
//
// Every routine is the definition written out as loops over the window; the only
// alternative form is normconv(direct=0), which evaluates the SAME double sum
// row-then-column (G(i,j) = g_i g_j, eq. 2) so that whole 1024^2 frames finish in
// seconds; tests/test_oracle_pins.py pins it to the direct form.
//
// Parity status: every function below is pinned by tests/test_oracle_*.py
// (closed forms, SciPy special cases, invariants, hand examples, injected
// sources).  "parity unpinned": only the *values chosen* for the free parameters
// the paper leaves open (s_bg / K, r_flux, r_dedupe, r_assoc, n_forget) -- any
// value is "correct"; they are parameters, not results.
// ---------------------------------------------------------------------------
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>

extern "C" {

// ---- O1: per-band statistics over valid pixels -----------------------------
// PAPER.md:377 (App. A): b = per-band image mean.  rms and one clip round are the
// north_star's "robust RMS" terms (R13).  stats[b] = {n, mean, rms,
// n_clip, clipped mean, clipped rms}; population (1/n) moments.
void orc_band_stats(const float* cube, int B, int Dy, int Dx, const uint8_t* W,
                    double qc_clip, double* stats) {
  const int64_t N = (int64_t)Dy * Dx;
  for (int b = 0; b < B; ++b) {
    const float* X = cube + (int64_t)b * N;
    double n = 0, sum = 0;
    for (int64_t i = 0; i < N; ++i)
      if (!W || W[i]) { n += 1; sum += (double)X[i]; }
    double* o = stats + 6 * b;
    if (n == 0) { for (int j = 0; j < 6; ++j) o[j] = 0; continue; }
    const double mean = sum / n;
    double ss = 0;
    for (int64_t i = 0; i < N; ++i)
      if (!W || W[i]) { double d = (double)X[i] - mean; ss += d * d; }
    const double rms = std::sqrt(ss / n);
    // one clip round, as defined (O1): the pixels with |x - mean| <= qc_clip rms, decided in float64 like
    // everything else here.  (A float32 implementation may put a pixel that sits within rounding of the
    // boundary on the other side; the parity harness classifies such pixels by THIS margin and logs them.)
    const double thr = qc_clip * rms;
    auto inside = [&](float x) { return std::fabs((double)x - mean) <= thr; };
    double nc = 0, sc = 0;
    for (int64_t i = 0; i < N; ++i)
      if ((!W || W[i]) && inside(X[i])) { nc += 1; sc += (double)X[i]; }
    double cmean = 0, crms = 0;
    if (nc > 0) {
      cmean = sc / nc;
      double ssc = 0;
      for (int64_t i = 0; i < N; ++i)
        if ((!W || W[i]) && inside(X[i])) { double e = (double)X[i] - cmean; ssc += e * e; }
      crms = std::sqrt(ssc / nc);
    }
    o[0] = n; o[1] = mean; o[2] = rms; o[3] = nc; o[4] = cmean; o[5] = crms;
  }
}

static double median_of(std::vector<double> v) {
  std::sort(v.begin(), v.end());
  const size_t m = v.size();
  if (m == 0) return 0.0;
  return (m & 1) ? v[m / 2] : 0.5 * (v[m / 2 - 1] + v[m / 2]);
}

// ---- O2: cross-band robust verdict ------------------------------------------
// PAPER.md:379 eq. A.1: z = (b - median(b)) / MAD(b), threshold "e.g. 5" (:381),
// rejected band == zero-imputed image (:387).  Readings: MAD = median
// absolute deviation, unscaled (R10); two-sided (R11); denominator floored at the
// standard error SE_mean = median(rms)/sqrt(n), SE_rms = median(rms)/sqrt(2n)
// (R12); applied to the mean vector AND the rms vector (R13); a band whose mean or
// rms is not finite (or n = 0) is rejected and left out of the medians;
// frame_ok = #ok >= ceil(B/2).   z[b] = {z_mean, z_rms};  band_ok[B] = frame_ok.
void orc_qc_verdict(const double* stats, int B, double tau, double* z, uint8_t* band_ok) {
  std::vector<int> fin;
  for (int b = 0; b < B; ++b) {
    const double* s = stats + 6 * b;
    if (s[0] > 0 && std::isfinite(s[1]) && std::isfinite(s[2])) fin.push_back(b);
  }
  for (int b = 0; b < B; ++b) { z[2 * b] = z[2 * b + 1] = std::numeric_limits<double>::infinity(); band_ok[b] = 0; }
  int n_ok = 0;
  if (!fin.empty()) {
    std::vector<double> vm, vr;
    for (int b : fin) { vm.push_back(stats[6 * b + 1]); vr.push_back(stats[6 * b + 2]); }
    const double med_m = median_of(vm), med_r = median_of(vr);
    std::vector<double> am, ar;
    for (size_t i = 0; i < fin.size(); ++i) { am.push_back(std::fabs(vm[i] - med_m)); ar.push_back(std::fabs(vr[i] - med_r)); }
    const double mad_m = median_of(am), mad_r = median_of(ar);
    for (size_t i = 0; i < fin.size(); ++i) {
      const int b = fin[i];
      const double n = stats[6 * b];
      const double den_m = std::max(mad_m, med_r / std::sqrt(n));
      const double den_r = std::max(mad_r, med_r / std::sqrt(2.0 * n));
      auto zz = [](double num, double den) {
        if (den > 0) return num / den;
        if (num == 0) return 0.0;
        return num > 0 ? std::numeric_limits<double>::infinity() : -std::numeric_limits<double>::infinity();
      };
      z[2 * b] = zz(vm[i] - med_m, den_m);
      z[2 * b + 1] = zz(vr[i] - med_r, den_r);
      band_ok[b] = (std::fabs(z[2 * b]) <= tau && std::fabs(z[2 * b + 1]) <= tau) ? 1 : 0;
      n_ok += band_ok[b];
    }
  }
  band_ok[B] = (n_ok >= (B + 1) / 2) ? 1 : 0;
}

// ---- O3: kernel taps ---------------------------------------------------------
// PAPER.md:74-77 eq. 2: G(n,m,s) = exp[-(n^2+m^2)/(2 s^2)] / Z with Z the sum over
// the (2k+1)^2 kernel offsets (R1), so G(i,j) = g_i g_j with
// g_i = e_i / sum_{|i|<=k} e_i.  kind 1: uniform ("a (circular) uniform kernel",
// :77; we take the square one) g_i = 1/(2k+1).  s <= 0 with kind 0: identity
// (g = delta), the paper-literal "no matched filter" mode.
void orc_kernel_taps(int kind, double s, int k, double* g) {
  const int n = 2 * k + 1;
  if (kind == 1) { for (int i = 0; i < n; ++i) g[i] = 1.0 / n; return; }
  if (s <= 0) { for (int i = 0; i < n; ++i) g[i] = (i == k) ? 1.0 : 0.0; return; }
  double sum = 0;
  for (int i = -k; i <= k; ++i) { g[i + k] = std::exp(-(double)(i * i) / (2.0 * s * s)); sum += g[i + k]; }
  for (int i = 0; i < n; ++i) g[i] /= sum;
}

// ---- normalised convolution (eq. 3 with borders / mask / clipped pixels) -----
// (g (*)_Wp A)(n,m) = sum_{|i|,|j|<=k, in image} g_i g_j Wp A / sum g_i g_j Wp,
// 0 where the denominator is 0 (R6, R7).  In the interior with Wp == 1 the
// denominator is 1 and this is eq. 3's plain G*X.
// direct = 1: the 2-D window sum as written.  direct = 0: same sum, rows then
// columns.  Wp == NULL means all ones.  `den_out` (optional) receives the
// denominator.
void orc_normconv(const double* A, const uint8_t* Wp, int Dy, int Dx, const double* g, int k,
                  int direct, double* out, double* den_out) {
  const int64_t N = (int64_t)Dy * Dx;
  if (direct) {
    for (int y = 0; y < Dy; ++y)
      for (int x = 0; x < Dx; ++x) {
        double num = 0, den = 0;
        for (int j = -k; j <= k; ++j) {
          const int yy = y + j;
          if (yy < 0 || yy >= Dy) continue;
          for (int i = -k; i <= k; ++i) {
            const int xx = x + i;
            if (xx < 0 || xx >= Dx) continue;
            const int64_t q = (int64_t)yy * Dx + xx;
            if (Wp && !Wp[q]) continue;
            const double w = g[j + k] * g[i + k];
            num += w * A[q];
            den += w;
          }
        }
        const int64_t p = (int64_t)y * Dx + x;
        out[p] = den > 0 ? num / den : 0.0;
        if (den_out) den_out[p] = den;
      }
    return;
  }
  std::vector<double> rn(N), rd(N);
  for (int y = 0; y < Dy; ++y)
    for (int x = 0; x < Dx; ++x) {
      double num = 0, den = 0;
      for (int i = -k; i <= k; ++i) {
        const int xx = x + i;
        if (xx < 0 || xx >= Dx) continue;
        const int64_t q = (int64_t)y * Dx + xx;
        if (Wp && !Wp[q]) continue;
        num += g[i + k] * A[q];
        den += g[i + k];
      }
      rn[(int64_t)y * Dx + x] = num; rd[(int64_t)y * Dx + x] = den;
    }
  for (int y = 0; y < Dy; ++y)
    for (int x = 0; x < Dx; ++x) {
      double num = 0, den = 0;
      for (int j = -k; j <= k; ++j) {
        const int yy = y + j;
        if (yy < 0 || yy >= Dy) continue;
        const int64_t q = (int64_t)yy * Dx + x;
        num += g[j + k] * rn[q];
        den += g[j + k] * rd[q];
      }
      const int64_t p = (int64_t)y * Dx + x;
      out[p] = den > 0 ? num / den : 0.0;
      if (den_out) den_out[p] = den;
    }
}

// ---- O4: planes --------------------------------------------------------------
// Plane p < B is band p (all zero if rejected: "imputing the entire image with
// zeros"); plane B is the sum over accepted bands (north_star; the
// paper only discusses it as eq. B.7, R5).  planes: [B+1][Dy][Dx] float64.
void orc_planes(const float* cube, const uint8_t* band_ok, int B, int Dy, int Dx, double* planes) {
  const int64_t N = (int64_t)Dy * Dx;
  double* sum = planes + (int64_t)B * N;
  for (int64_t i = 0; i < N; ++i) sum[i] = 0;
  for (int b = 0; b < B; ++b) {
    double* P = planes + (int64_t)b * N;
    const float* X = cube + (int64_t)b * N;
    if (band_ok[b]) { for (int64_t i = 0; i < N; ++i) { P[i] = (double)X[i]; sum[i] += (double)X[i]; } }
    else            { for (int64_t i = 0; i < N; ++i) P[i] = 0.0; }
  }
}

// ---- O4-O6 for one plane: matched filter, clip loop, local maxima ------------
// F = g_mf (*)_W X, 0 where W = 0                                  (eq. 2 kernel; R4)
// for it = 1..n_iter:  W' = W and not Y                             (R6)
//   C = g_bg (*)_{W'} F                                             (eq. 3)
//   S = g_bg (*)_{W'} (F - C)^2      square at the same pixel       (eq. 4)
//   S_eff = max(S, (eps_rel |C|)^2)                                 (R8)
//   new = not Y and W and F-C > 0 and (F-C)^2 > kappa^2 S_eff       (eq. 5)
//   Y |= new                          (until no new y or a fixed count)
// Q = [F >= F(i,j) for all valid in-image (i,j) in the (2 k_max+1)^2 window]
//                                                                   (eq. 6; R9)
// P = Q and Y                                                       (eq. 7)
// Outputs (all [Dy][Dx]): F; iter (uint8: 0 = never, else iteration of first
// detection); at first detection C, S_eff, snr = (F-C)/sqrt(S_eff); Q, P (uint8).
// C_last / S_last (optional): C and raw S of the LAST iteration, every pixel.
void orc_detect_plane(const double* X, const uint8_t* W, int Dy, int Dx,
                      const double* g_mf, int k_mf, const double* g_bg, int k_bg,
                      double kappa, double eps_rel, int n_iter, int k_max, int direct,
                      double* F, uint8_t* iter, double* Cdet, double* Sdet, double* snr,
                      uint8_t* Q, uint8_t* P, double* C_last, double* S_last) {
  const int64_t N = (int64_t)Dy * Dx;
  orc_normconv(X, W, Dy, Dx, g_mf, k_mf, direct, F, nullptr);
  for (int64_t i = 0; i < N; ++i) { if (W && !W[i]) F[i] = 0.0; iter[i] = 0; Cdet[i] = Sdet[i] = snr[i] = 0.0; }
  std::vector<uint8_t> Wp(N);
  std::vector<double> C(N), R(N), S(N);
  for (int it = 1; it <= n_iter; ++it) {
    for (int64_t i = 0; i < N; ++i) Wp[i] = ((!W || W[i]) && !iter[i]) ? 1 : 0;
    orc_normconv(F, Wp.data(), Dy, Dx, g_bg, k_bg, direct, C.data(), nullptr);
    for (int64_t i = 0; i < N; ++i) { const double d = F[i] - C[i]; R[i] = d * d; }
    orc_normconv(R.data(), Wp.data(), Dy, Dx, g_bg, k_bg, direct, S.data(), nullptr);
    int64_t n_new = 0;
    for (int64_t i = 0; i < N; ++i) {
      if (iter[i] || (W && !W[i])) continue;
      const double d = F[i] - C[i];
      const double guard = eps_rel * std::fabs(C[i]);
      const double se = std::max(S[i], guard * guard);
      if (d > 0 && d * d > kappa * kappa * se) {
        iter[i] = (uint8_t)it; Cdet[i] = C[i]; Sdet[i] = se; snr[i] = d / std::sqrt(se); ++n_new;
      }
    }
    if (it == n_iter || n_new == 0) {
      if (C_last) std::memcpy(C_last, C.data(), N * sizeof(double));
      if (S_last) std::memcpy(S_last, S.data(), N * sizeof(double));
    }
    if (n_new == 0) break;  // "until no new y_nm is discovered" -- same result as running on
  }
  for (int y = 0; y < Dy; ++y)
    for (int x = 0; x < Dx; ++x) {
      const int64_t p = (int64_t)y * Dx + x;
      uint8_t q = 0;
      if (!W || W[p]) {
        q = 1;
        for (int j = -k_max; j <= k_max && q; ++j) {
          const int yy = y + j;
          if (yy < 0 || yy >= Dy) continue;
          for (int i = -k_max; i <= k_max; ++i) {
            const int xx = x + i;
            if (xx < 0 || xx >= Dx) continue;
            const int64_t r = (int64_t)yy * Dx + xx;
            if (W && !W[r]) continue;
            if (F[r] > F[p]) { q = 0; break; }
          }
        }
      }
      Q[p] = q;
      P[p] = (q && iter[p]) ? 1 : 0;
    }
}

// ---- O7: cross-plane duplicate filter ----------------------------------------
// "we filter the duplicates that we obtain from measuring at different
// frequencies simultaneously" (no algorithm given -> R17):
// M(pix) = max over planes with P = 1 of snr (ties -> lowest plane); a pixel is
// kept iff no OTHER pixel within Euclidean distance r_dedupe carries a
// lexicographically larger (M, -pix).  One shot, order independent.
// Input: n records (pix, plane, snr) in any order.  Output sorted by pix.
int orc_dedupe(const int32_t* pix, const int16_t* plane, const double* snr, int n,
               int Dy, int Dx, int r_dedupe,
               int32_t* upos, int16_t* uplane, double* usnr) {
  struct E { int32_t pix; int16_t plane; double m; };
  std::vector<E> best;
  {
    std::vector<int> order(n);
    for (int i = 0; i < n; ++i) order[i] = i;
    std::sort(order.begin(), order.end(), [&](int a, int b) { return pix[a] != pix[b] ? pix[a] < pix[b] : plane[a] < plane[b]; });
    for (int oi = 0; oi < n; ++oi) {
      const int i = order[oi];
      if (best.empty() || best.back().pix != pix[i]) best.push_back({pix[i], plane[i], snr[i]});
      else if (snr[i] > best.back().m) { best.back().m = snr[i]; best.back().plane = plane[i]; }
    }
  }
  int nu = 0;
  for (size_t a = 0; a < best.size(); ++a) {
    const int ya = best[a].pix / Dx, xa = best[a].pix % Dx;
    bool keep = true;
    for (size_t b = 0; b < best.size() && keep; ++b) {
      if (a == b) continue;
      const int yb = best[b].pix / Dx, xb = best[b].pix % Dx;
      const int dy = ya - yb, dx = xa - xb;
      if (dy * dy + dx * dx > r_dedupe * r_dedupe) continue;
      if (best[b].m > best[a].m || (best[b].m == best[a].m && best[b].pix < best[a].pix)) keep = false;
    }
    if (keep) { upos[nu] = best[a].pix; uplane[nu] = best[a].plane; usnr[nu] = best[a].m; ++nu; }
  }
  (void)Dy;
  return nu;
}

// ---- O8: association with the t-1 catalogue, monitoring ----------------------
// match to the previous time-step's sources by 2-D distance within a
// limit; keep monitoring until not detected for a pre-specified number of steps.
// Readings (R16, R17): pixel distance d^2 <= r_assoc^2 against the table as it was
// BEFORE this frame; nearest wins, tie -> lowest slot; a candidate keeps the pixel
// of its first detection; unmatched candidates age by one ACCEPTED frame and are
// retired at miss >= n_forget (forced candidates never); then unmatched
// detections, in ascending pix, take the lowest free slots; no free slot ->
// cand_idx = -1 and *n_dropped += 1.  frame_ok = 0: nothing changes.
// Table arrays (length n_cand_max): active (u8), forced (u8), cpix (i32),
// miss (i32), born (i64).  Outputs: cand_idx[nu]; act_slots/act_pix (ascending
// slot) and the return value = number of active slots after this frame.
int orc_associate(uint8_t* active, uint8_t* forced, int32_t* cpix, int32_t* miss, int64_t* born,
                  int n_cand_max, const int32_t* upos, int nu, int64_t t, int frame_ok,
                  int Dx, int r_assoc, int n_forget,
                  int32_t* cand_idx, int32_t* act_slots, int32_t* act_pix, int32_t* n_dropped) {
  if (frame_ok) {
    std::vector<uint8_t> matched(n_cand_max, 0);
    for (int i = 0; i < nu; ++i) {
      const int y = upos[i] / Dx, x = upos[i] % Dx;
      long best_d = -1; int best_s = -1;
      for (int s = 0; s < n_cand_max; ++s) {
        if (!active[s]) continue;
        const int dy = y - cpix[s] / Dx, dx = x - cpix[s] % Dx;
        const long d2 = (long)dy * dy + (long)dx * dx;
        if (d2 > (long)r_assoc * r_assoc) continue;
        if (best_s < 0 || d2 < best_d) { best_d = d2; best_s = s; }
      }
      cand_idx[i] = best_s;
    }
    for (int i = 0; i < nu; ++i) if (cand_idx[i] >= 0) matched[cand_idx[i]] = 1;
    for (int s = 0; s < n_cand_max; ++s) {
      if (!active[s]) continue;
      if (matched[s]) miss[s] = 0;
      else { miss[s] += 1; if (!forced[s] && miss[s] >= n_forget) active[s] = 0; }
    }
    int s_free = 0;
    for (int i = 0; i < nu; ++i) {
      if (cand_idx[i] >= 0) continue;
      while (s_free < n_cand_max && active[s_free]) ++s_free;
      if (s_free >= n_cand_max) { cand_idx[i] = -1; if (n_dropped) *n_dropped += 1; continue; }
      active[s_free] = 1; forced[s_free] = 0; cpix[s_free] = upos[i]; miss[s_free] = 0; born[s_free] = t;
      cand_idx[i] = s_free;
    }
  } else {
    for (int i = 0; i < nu; ++i) cand_idx[i] = -1;
  }
  int na = 0;
  for (int s = 0; s < n_cand_max; ++s) if (active[s]) { act_slots[na] = s; act_pix[na] = cpix[s]; ++na; }
  return na;
}

// ---- O9: forced peak flux -----------------------------------------------------
// "taking the maximum pixel value within a box around the source peak ... at all
// frequencies".  Box half-width r_flux (R15), raw cube, valid
// in-image pixels only; rejected band (or rejected frame) -> 0 (zero-imputed
// image); no valid pixel in the box -> 0.  flux: [npos][B] float32
// (a max of float32 inputs: exact).
void orc_measure_flux(const float* cube, const uint8_t* band_ok, const uint8_t* W, int B, int Dy, int Dx,
                      const int32_t* pos, int npos, int r_flux, float* flux) {
  const int64_t N = (int64_t)Dy * Dx;
  const int frame_ok = band_ok[B];
  for (int i = 0; i < npos; ++i) {
    const int y = pos[i] / Dx, x = pos[i] % Dx;
    for (int b = 0; b < B; ++b) {
      float best = 0.0f; bool any = false;
      if (frame_ok && band_ok[b]) {
        for (int j = -r_flux; j <= r_flux; ++j) {
          const int yy = y + j; if (yy < 0 || yy >= Dy) continue;
          for (int k = -r_flux; k <= r_flux; ++k) {
            const int xx = x + k; if (xx < 0 || xx >= Dx) continue;
            const int64_t q = (int64_t)yy * Dx + xx;
            if (W && !W[q]) continue;
            const float v = cube[(int64_t)b * N + q];
            if (!any || v > best) { best = v; any = true; }
          }
        }
      }
      flux[(int64_t)i * B + b] = any ? best : 0.0f;
    }
  }
}

// ---- O10: dynamic-spectrum ring buffers ---------------------------------------
// "Collecting the fluxes over time at different bandpasses yields dynamic spectra"
// (Fig. 1 :23).  ring[slot][t mod T_ring][b]; a slot born at t is
// pre-filled with NaN first; meta_t[tau] = t, meta_ok[tau] = band_ok bits.
void orc_ring_append(float* ring, int64_t* meta_t, uint64_t* meta_ok, const int64_t* born,
                     int T_ring, int B, const int32_t* slots, int n, const float* flux,
                     const uint8_t* band_ok, int64_t t) {
  const int tau = (int)(t % T_ring);
  for (int i = 0; i < n; ++i) {
    const int s = slots[i];
    float* r = ring + (int64_t)s * T_ring * B;
    if (born[s] == t)
      for (int64_t q = 0; q < (int64_t)T_ring * B; ++q) r[q] = std::numeric_limits<float>::quiet_NaN();
    for (int b = 0; b < B; ++b) r[(int64_t)tau * B + b] = flux[(int64_t)i * B + b];
  }
  meta_t[tau] = t;
  uint64_t bits = 0;
  for (int b = 0; b < B && b < 64; ++b) if (band_ok[B] && band_ok[b]) bits |= (1ull << b);
  meta_ok[tau] = bits;
}

// Time-ordered frequency x time view of one slot, oldest -> newest, ending at
// t_last: out[b][j] is the sample of time t_last - T_ring + 1 + j, NaN where that
// time was never appended (meta_t mismatch) or precedes the slot's birth.
void orc_get_dynspec(const float* ring, const int64_t* meta_t, int T_ring, int B, int slot,
                     int64_t t_last, float* out) {
  const float* r = ring + (int64_t)slot * T_ring * B;
  for (int j = 0; j < T_ring; ++j) {
    const int64_t tt = t_last - T_ring + 1 + j;
    const int tau = (int)(((tt % T_ring) + T_ring) % T_ring);
    const bool have = tt >= 0 && meta_t[tau] == tt;
    for (int b = 0; b < B; ++b)
      out[(int64_t)b * T_ring + j] = have ? r[(int64_t)tau * B + b] : std::numeric_limits<float>::quiet_NaN();
  }
}

int orc_version(void) { return 1; }

}  // extern "C"
