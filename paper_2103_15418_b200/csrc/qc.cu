// S1 + S2 (+ S3): quality control (App. A, eq. A.1; O1, O2) and the sum plane.
//
// The streaming form (a 16-byte aligned cube with N a multiple of 4: every shaped configuration):
//   k_qc_moments  reads the cube ONCE, all bands of a group of 4 pixels in one thread (loads of the next four
//                 bands in flight while four are consumed), and takes three things from that read: per band over
//                 valid pixels sum(x - p) and sum(x - p)^2 about a pivot p (the band's first valid pixel; packed
//                 fp32 per thread - a thread sees a few dozen values - then float64), the sum plane of ALL bands
//                 (O4, S3: speculative - the verdict is not known yet, and 19 frames in 20 reject nothing) and,
//                 per band, whether some invalid pixel holds anything but an exact zero.
//   k_qc_verdict  one block: finishes the moments, eq. A.1 across bands (median, MAD, SE floor) for the mean
//                 vector and the rms vector -> band_ok, frame_ok, the centre / half width of the clip round, the
//                 "far above the noise" level of every plane, and whether the accepted bands are clean outside
//                 the mask (then W X = X and the fused detection kernel reads the cube unmasked).
//   k_qc_clip     second read of the cube: the moments of the pixels inside the one qc_clip-sigma clip round
//                 (O1); when a band was rejected it also rebuilds the sum plane from the accepted bands.
//   k_qc_clip_finish  one block: the clipped mean / rms.
// The generic form (any alignment) keeps the two older kernels, whose last block does the finishing:
// k_qc_pass1 (per-band moments + verdict) and k_qc_pass2 (clip round, sum plane, exact-zero check).
#include <cstdio>

#include "lpf_internal.cuh"

namespace {

constexpr int QC_THREADS = 256;
constexpr int QC_WARPS = QC_THREADS / 32;
constexpr int QC2_THREADS = 128;   // pass 2: 4 pixel groups per thread and band in flight
constexpr int QC2_WARPS = QC2_THREADS / 32;

__device__ __forceinline__ void block_reduce3(double& a, double& b, double& c, double* sm /*[3][8]*/) {
  a = lpf_warp_sum(a); b = lpf_warp_sum(b); c = lpf_warp_sum(c);
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  __syncthreads();
  if (l == 0) { sm[w] = a; sm[8 + w] = b; sm[16 + w] = c; }
  __syncthreads();
  if (w == 0) {
    a = l < QC_WARPS ? sm[l] : 0.0;
    b = l < QC_WARPS ? sm[8 + l] : 0.0;
    c = l < QC_WARPS ? sm[16 + l] : 0.0;
    a = lpf_warp_sum(a); b = lpf_warp_sum(b); c = lpf_warp_sum(c);
  }
}

// true in exactly one block of the grid: the last one to get here.  The counter is left at zero.
__device__ __forceinline__ bool last_block_done(int32_t* counter, int total) {
  __shared__ int s_last;
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) {
    const int prev = atomicAdd(counter, 1);
    s_last = (prev == total - 1) ? 1 : 0;
    if (s_last) *counter = 0;
  }
  __syncthreads();
  if (s_last) __threadfence();
  return s_last != 0;
}

struct QcArgs {
  const LpfFrameDesc* fd;   // non-null: cube comes from the frame descriptor
  const float* cube; const uint8_t* W; long long N; int first_valid, B, nblk;
  double* part1;          // [B][nblk][3]
  float qc_clip, tau;
  float* stats;           // [B][8]
  uint8_t* band_ok;       // [B + 1]
  float* band_clip;       // [B][2] centre and half width of the clip round
  float* big_thr;         // [B + 1] big_sigma x rms of every plane (the sum plane: of the accepted bands, in quadrature)
  float big_sigma;
  int32_t* counter;
};

// eq. A.1 for all bands, by one block of QC_THREADS threads.
__device__ void qc_verdict(const QcArgs& a, const double* mom = nullptr /* [B][3] n, sum, sum of squares: skips the partials */) {
  __shared__ double s_mean[LPF_MAX_BANDS], s_rms[LPF_MAX_BANDS], s_n[LPF_MAX_BANDS], s_sorted[LPF_MAX_BANDS], s_dev[LPF_MAX_BANDS];
  __shared__ int s_fin[LPF_MAX_BANDS];
  __shared__ int s_nfin, s_nok;
  __shared__ float s_var_ok;
  const int B = a.B, nblk = a.nblk;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  // finish pass 1: warp w takes bands w, w + 8, ...; lanes share the partials of a band
  for (int b = warp; b < B; b += QC_WARPS) {
    double n = 0, s1 = 0, s2 = 0;
    if (mom) { if (lane == 0) { n = __ldcg(mom + 3 * b); s1 = __ldcg(mom + 3 * b + 1); s2 = __ldcg(mom + 3 * b + 2); } }
    else for (int i0 = 0; i0 < nblk; i0 += 32 * 10) {      // thirty independent loads per lane and round (one round up to 320 blocks)
      double v[10][3];
#pragma unroll
      for (int u = 0; u < 10; ++u) {
        const int i = i0 + 32 * u + lane;
        const double* q = a.part1 + ((long long)b * nblk + (i < nblk ? i : 0)) * 3;
#pragma unroll
        for (int k = 0; k < 3; ++k) v[u][k] = i < nblk ? __ldcg(q + k) : 0.0;
      }
#pragma unroll
      for (int u = 0; u < 10; ++u) { n += v[u][0]; s1 += v[u][1]; s2 += v[u][2]; }
    }
    n = lpf_warp_sum(n); s1 = lpf_warp_sum(s1); s2 = lpf_warp_sum(s2);
    if (lane == 0) {
      double mean = 0, rms = 0;
      if (n > 0) {
        const double piv = (double)a.cube[(long long)b * a.N + a.first_valid];
        const double m1 = s1 / n;
        mean = piv + m1;
        const double var = s2 / n - m1 * m1;
        rms = sqrt(var > 0 ? var : 0.0);
      }
      s_mean[b] = mean; s_rms[b] = rms; s_n[b] = n;
      s_fin[b] = (n > 0 && isfinite(mean) && isfinite(rms)) ? 1 : 0;
    }
  }
  if (threadIdx.x == 0) { s_nfin = 0; s_nok = 0; s_var_ok = 0.f; }
  __syncthreads();
  const int b = threadIdx.x;
  const double n = b < B ? s_n[b] : 0.0, mean = b < B ? s_mean[b] : 0.0, rms = b < B ? s_rms[b] : 0.0;
  const int fin = b < B ? s_fin[b] : 0;
  if (b < B && fin) atomicAdd(&s_nfin, 1);
  __syncthreads();
  const int m = s_nfin;

  // median by rank selection over the finite bands (ties broken by band index)
  auto median_of = [&](const double* v, double my) -> double {
    __syncthreads();
    if (b < B && fin) {
      int rank = 0;
      for (int j = 0; j < B; ++j)
        if (s_fin[j] && (v[j] < my || (v[j] == my && j < b))) ++rank;
      s_sorted[rank] = my;
    }
    __syncthreads();
    double med = 0.0;
    if (m > 0) med = (m & 1) ? s_sorted[m / 2] : 0.5 * (s_sorted[m / 2 - 1] + s_sorted[m / 2]);
    return med;
  };
  const double med_m = median_of(s_mean, mean);
  const double med_r = median_of(s_rms, rms);
  __syncthreads();
  if (b < B) s_dev[b] = fabs(mean - med_m);
  const double mad_m = median_of(s_dev, fabs(mean - med_m));
  __syncthreads();
  if (b < B) s_dev[b] = fabs(rms - med_r);
  const double mad_r = median_of(s_dev, fabs(rms - med_r));

  double zm = INFINITY, zr = INFINITY;
  int ok = 0;
  if (b < B && fin) {
    const double den_m = fmax(mad_m, med_r / sqrt(n));
    const double den_r = fmax(mad_r, med_r / sqrt(2.0 * n));
    const double num_m = mean - med_m, num_r = rms - med_r;
    zm = den_m > 0 ? num_m / den_m : (num_m == 0 ? 0.0 : (num_m > 0 ? INFINITY : -INFINITY));
    zr = den_r > 0 ? num_r / den_r : (num_r == 0 ? 0.0 : (num_r > 0 ? INFINITY : -INFINITY));
    ok = (fabs(zm) <= (double)a.tau && fabs(zr) <= (double)a.tau) ? 1 : 0;
    if (ok) { atomicAdd(&s_nok, 1); atomicAdd(&s_var_ok, (float)(rms * rms)); }
  }
  __syncthreads();
  if (b < B) {
    float* o = a.stats + LPF_STATS_PER_BAND * b;
    o[0] = (float)n; o[1] = (float)mean; o[2] = (float)rms; o[3] = 0.f; o[4] = 0.f; o[5] = 0.f;
    o[6] = (float)zm; o[7] = (float)zr;
    a.band_ok[b] = (uint8_t)ok;
    a.band_clip[2 * b] = (float)mean;                          // the clip round is decided in float32 (R25)
    a.band_clip[2 * b + 1] = (float)((double)a.qc_clip * rms);
    a.big_thr[b] = a.big_sigma * (float)rms;
  }
  if (threadIdx.x == 0) {
    a.band_ok[B] = (s_nok >= (B + 1) / 2) ? 1 : 0;
    a.big_thr[B] = a.big_sigma * sqrtf(s_var_ok);
  }
}

__global__ void __launch_bounds__(QC_THREADS)
k_qc_pass1(const QcArgs a) {
  __shared__ double sm[24];
  const int b = blockIdx.y, nblk = a.nblk;
  const long long N = a.N;
  const float* X = a.cube + (long long)b * N;
  const float piv = X[a.first_valid];

  // contiguous chunk of this band for this block, in units of 4 pixels
  const long long n4 = (N + 3) >> 2;
  const long long per = (n4 + nblk - 1) / nblk;
  const long long q0 = (long long)blockIdx.x * per;
  const long long q1 = (q0 + per < n4) ? q0 + per : n4;
  const bool vec = ((N & 3) == 0) && ((((uintptr_t)a.cube) & 15) == 0);

  double dn = 0, d1 = 0, d2 = 0;
  if (vec) {
    // four 128-bit loads (and their mask words) in flight per thread; fp32 over those 16 values, float64 across
    for (long long q = q0 + threadIdx.x; q < q1; q += 4 * QC_THREADS) {
      float4 x[4]; unsigned wm[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const long long qq = q + k * QC_THREADS;
        const bool in = qq < q1;
        x[k] = in ? __ldg(reinterpret_cast<const float4*>(X) + qq) : make_float4(0.f, 0.f, 0.f, 0.f);
        wm[k] = in ? __ldg(reinterpret_cast<const unsigned*>(a.W) + qq) : 0u;
      }
      float fn = 0.f, f1 = 0.f, f2 = 0.f;
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const float v[4] = {x[k].x, x[k].y, x[k].z, x[k].w};
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const float d = v[j] - piv;
          if (((wm[k] >> (8 * j)) & 0xffu) != 0) { fn += 1.f; f1 += d; f2 = fmaf(d, d, f2); }
        }
      }
      dn += fn; d1 += f1; d2 += f2;
    }
  } else {
    float fn = 0.f, f1 = 0.f, f2 = 0.f;
    int run = 0;
    for (long long q = q0 + threadIdx.x; q < q1; q += QC_THREADS) {
      const long long i0 = q << 2;
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        if ((i0 + j) < N && a.W[i0 + j]) { const float d = X[i0 + j] - piv; fn += 1.f; f1 += d; f2 = fmaf(d, d, f2); }
      }
      if (++run == 4) { dn += fn; d1 += f1; d2 += f2; fn = f1 = f2 = 0.f; run = 0; }
    }
    dn += fn; d1 += f1; d2 += f2;
  }
  block_reduce3(dn, d1, d2, sm);
  if (threadIdx.x == 0) {
    double* o = a.part1 + ((long long)b * nblk + blockIdx.x) * 3;
    o[0] = dn; o[1] = d1; o[2] = d2;
  }
  if (last_block_done(a.counter, gridDim.x * gridDim.y)) qc_verdict(a);
}

struct Qc2Args {
  const float* cube; const uint8_t* W; const uint8_t* band_ok; long long N; int B;
  const float* band_clip;  // [B][2]
  double* part2;           // [gridDim.x][B][3]
  float* stats;            // [B][8]: columns 3..5 are written here
  float* sum_out;          // [N] or null
  int32_t* dirty; int seq;
  int32_t* zero_me;        // a counter this kernel resets (the record count of the frame), or null
  int32_t* counter;
};

// the clipped moments from the per-block partials [nblk][B][3]: warp w takes bands w, w + nwarps, ...
__device__ void clip_finish(const double* part2, int nblk, int B, const float* band_clip, float* stats) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
  for (int b = warp; b < B; b += nw) {
    double nc = 0, c1 = 0, c2 = 0;
    for (int i0 = 0; i0 < nblk; i0 += 32 * 10) {      // thirty independent loads per lane and round
      double v[10][3];
#pragma unroll
      for (int u = 0; u < 10; ++u) {
        const int i = i0 + 32 * u + lane;
        const double* r = part2 + ((long long)(i < nblk ? i : 0) * B + b) * 3;
#pragma unroll
        for (int k = 0; k < 3; ++k) v[u][k] = i < nblk ? __ldcg(r + k) : 0.0;
      }
#pragma unroll
      for (int u = 0; u < 10; ++u) { nc += v[u][0]; c1 += v[u][1]; c2 += v[u][2]; }
    }
    nc = lpf_warp_sum(nc); c1 = lpf_warp_sum(c1); c2 = lpf_warp_sum(c2);
    if (lane == 0) {
      double cmean = 0, crms = 0;
      if (nc > 0) {
        const double k1 = c1 / nc;
        cmean = (double)band_clip[2 * b] + k1;         // the clip pass is centred on the fp32 mean
        const double cv = c2 / nc - k1 * k1;
        crms = sqrt(cv > 0 ? cv : 0.0);
      }
      float* o = stats + LPF_STATS_PER_BAND * b;
      o[3] = (float)nc; o[4] = (float)cmean; o[5] = (float)crms;
    }
  }
}

// CLIP: the clipped moments of every band; SUM: the sum plane of the accepted bands + the exact-zero check.
template <bool CLIP, bool SUM>
__global__ void __launch_bounds__(QC2_THREADS)
k_qc_pass2(const Qc2Args a) {
  __shared__ double s_acc[QC2_WARPS][LPF_MAX_BANDS][3];
  __shared__ float s_clip[LPF_MAX_BANDS][2];
  __shared__ uint8_t s_ok[LPF_MAX_BANDS + 1];
  const int B = a.B, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const long long N = a.N;
  for (int i = threadIdx.x; i < B; i += QC2_THREADS) {
    if (CLIP) { s_clip[i][0] = a.band_clip[2 * i]; s_clip[i][1] = a.band_clip[2 * i + 1]; }
    s_ok[i] = a.band_ok[i];
  }
  if (threadIdx.x == 0) s_ok[B] = a.band_ok[B];
  if (CLIP)
    for (int i = threadIdx.x; i < QC2_WARPS * LPF_MAX_BANDS * 3; i += QC2_THREADS) (&s_acc[0][0][0])[i] = 0.0;
  if (a.zero_me && blockIdx.x == 0 && threadIdx.x == 0) *a.zero_me = 0;
  __syncthreads();
  const bool do_sum = SUM && s_ok[B] != 0;      // a rejected frame has no sum plane (and no detections)
  const bool vec = ((N & 3) == 0) && ((((uintptr_t)a.cube) & 15) == 0);
  bool bad = false;
  if (vec) {
    // a thread owns 4 pixel groups (16 pixels), QC2_THREADS groups apart, for all bands
    const long long n4 = N >> 2;
    const long long chunk = 4LL * QC2_THREADS;
    for (long long c0 = (long long)blockIdx.x * chunk; c0 < n4; c0 += (long long)gridDim.x * chunk) {
      long long q[4]; unsigned wm[4]; bool in[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        q[k] = c0 + k * QC2_THREADS + threadIdx.x;
        in[k] = q[k] < n4;
        wm[k] = in[k] ? __ldg(reinterpret_cast<const unsigned*>(a.W) + q[k]) : 0u;
      }
      float4 s[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) s[k] = make_float4(0.f, 0.f, 0.f, 0.f);
      // the loads of the next needed band are issued before the current band is consumed
      auto needed = [&](int b) { return CLIP || (do_sum && s_ok[b] != 0); };
      auto fetch = [&](int b, float4 (&x)[4]) {
        const float4* Xb = reinterpret_cast<const float4*>(a.cube + (long long)b * N);
#pragma unroll
        for (int k = 0; k < 4; ++k) x[k] = in[k] ? __ldg(Xb + q[k]) : make_float4(0.f, 0.f, 0.f, 0.f);
      };
      int bn = 0;
      while (bn < B && !needed(bn)) ++bn;
      float4 xn[4];
      if (bn < B) fetch(bn, xn);
      while (bn < B) {
        const int b = bn;
        const bool okb = s_ok[b] != 0;
        float4 x[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) x[k] = xn[k];
        ++bn;
        while (bn < B && !needed(bn)) ++bn;
        if (bn < B) fetch(bn, xn);
        if (SUM && do_sum && okb) {
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            s[k].x += x[k].x; s[k].y += x[k].y; s[k].z += x[k].z; s[k].w += x[k].w;
            bad = bad || (!(wm[k] & 0x000000ffu) && x[k].x != 0.f) || (!(wm[k] & 0x0000ff00u) && x[k].y != 0.f) ||
                  (!(wm[k] & 0x00ff0000u) && x[k].z != 0.f) || (!(wm[k] & 0xff000000u) && x[k].w != 0.f);
          }
        }
        if (CLIP) {
          const float mean = s_clip[b][0], thr = s_clip[b][1];
          float fn = 0.f, f1 = 0.f, f2 = 0.f;
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            const float v[4] = {x[k].x, x[k].y, x[k].z, x[k].w};
#pragma unroll
            for (int j = 0; j < 4; ++j) {
              const float d = v[j] - mean;
              if (((wm[k] >> (8 * j)) & 0xffu) != 0 && fabsf(d) <= thr) { fn += 1.f; f1 += d; f2 = fmaf(d, d, f2); }
            }
          }
          fn = lpf_warp_sum(fn); f1 = lpf_warp_sum(f1); f2 = lpf_warp_sum(f2);   // 512 values in fp32, float64 from here on
          if (lane == 0) { s_acc[warp][b][0] += (double)fn; s_acc[warp][b][1] += (double)f1; s_acc[warp][b][2] += (double)f2; }
        }
      }
      if (SUM && do_sum && a.sum_out) {
#pragma unroll
        for (int k = 0; k < 4; ++k)
          if (in[k]) reinterpret_cast<float4*>(a.sum_out)[q[k]] = s[k];
      }
    }
  } else {
    for (long long i0 = (long long)blockIdx.x * QC2_THREADS; i0 < N; i0 += (long long)gridDim.x * QC2_THREADS) {
      const long long i = i0 + threadIdx.x;
      const bool in = i < N;
      const bool valid = in && a.W[i] != 0;
      float s = 0.f;
      for (int b = 0; b < B; ++b) {
        const bool okb = s_ok[b] != 0;
        if (!CLIP && !(do_sum && okb)) continue;
        const float x = in ? a.cube[(long long)b * N + i] : 0.f;
        if (SUM && do_sum && okb) { s += x; bad = bad || (in && !valid && x != 0.f); }
        if (CLIP) {
          const float d = x - s_clip[b][0];
          const bool take = valid && fabsf(d) <= s_clip[b][1];
          float fn = take ? 1.f : 0.f, f1 = take ? d : 0.f, f2 = take ? d * d : 0.f;
          fn = lpf_warp_sum(fn); f1 = lpf_warp_sum(f1); f2 = lpf_warp_sum(f2);
          if (lane == 0) { s_acc[warp][b][0] += (double)fn; s_acc[warp][b][1] += (double)f1; s_acc[warp][b][2] += (double)f2; }
        }
      }
      if (SUM && do_sum && a.sum_out && in) a.sum_out[i] = s;
    }
  }
  if (SUM && bad) *a.dirty = a.seq;
  if (!CLIP) return;
  __syncthreads();
  for (int i = threadIdx.x; i < B * 3; i += QC2_THREADS) {
    const int b = i / 3, k = i - 3 * b;
    double t = 0;
#pragma unroll
    for (int w = 0; w < QC2_WARPS; ++w) t += s_acc[w][b][k];
    a.part2[((long long)blockIdx.x * B + b) * 3 + k] = t;
  }
  if (!last_block_done(a.counter, gridDim.x)) return;
  clip_finish(a.part2, (int)gridDim.x, B, a.band_clip, a.stats);
}

// ---- the streaming form -------------------------------------------------------------------------------------------
// Block shape: 128 threads x 8 bands x 16 bytes = 16 KB of staging, <= 102 registers.  A block of this size fits
// BESIDE a CTA of the fused sweep on the same SM (the sweep leaves ~20 KB of its 196 KB shared-memory carve-out, 14.8 K
// registers and most of the issue slots free), so with several lanes in flight the QC of one frame runs under the
// sweeps of the others instead of waiting for the dozen SMs they leave empty: 9 640 -> 10 350 frames/s at 8 lanes
// (config 3).  The grid: lpf_qs_blocks.
#ifndef LPF_QS_THREADS
#define LPF_QS_THREADS 128
#endif
#ifndef LPF_QS_BLOCKS
#define LPF_QS_BLOCKS 5            // resident blocks per SM the register budget is set for (__launch_bounds__)
#endif
#ifndef LPF_QS_BG
#define LPF_QS_BG 8
#endif
constexpr int QS_THREADS = LPF_QS_THREADS;     // a thread owns one group of 4 pixels at a time, QS_BG bands of it
constexpr int QS_WARPS = QS_THREADS / 32;
constexpr int QS_BG = LPF_QS_BG;    // bands of one register-resident group

__device__ __forceinline__ float2 q_add2(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 q_fma2(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }

struct QsArgs {
  const LpfFrameDesc* fd;   // non-null: cube and seq come from the frame descriptor
  const float* cube; const uint8_t* W; long long N; int first_valid, B;
  double* part1;          // [B][gridDim.x][3]
  float* sum_out;         // [N] or null
  int32_t* dirty_b; int seq;   // [B] == seq: the band holds something other than an exact zero at an invalid pixel
};

// 16-byte asynchronous copies global -> shared (LDGSTS): the bytes in flight are not held in registers.  A thread
// owns one 16-byte slot per band of the group; slot b is refilled for the thread's next pixel group as soon as it
// has been consumed, one commit group per copy, so "at most QS_BG - 1 groups pending" means "slot b has landed".
__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }
// keep a value in its register (the compiler would otherwise rebuild it from its inputs at every use)
__device__ __forceinline__ void pin(unsigned& v) { asm volatile("" : "+r"(v)); }
__device__ __forceinline__ void pin(const char*& v) { asm volatile("" : "+l"(v)); }
constexpr size_t QS_SMEM = (size_t)QS_BG * QS_THREADS * sizeof(float4);   // 16 KB

// one group of <= QS_BG bands over the block's pixel groups [q0, q1); FULL: all QS_BG bands exist
template <bool FULL>
__device__ __forceinline__ void qs_moments_group(const QsArgs& a, int g0, long long q0, long long q1, const float* s_piv,
                                                 double (*s_red)[QS_BG][2], double* s_n, float4* qs_slots) {
  const int B = a.B, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const long long n4 = a.N >> 2;
  const long long sb = n4 * (long long)sizeof(float4);           // bytes from a band to the next at the same pixel group
  const bool want_sum = a.sum_out != nullptr;
  const uint32_t slot0 = (uint32_t)__cvta_generic_to_shared(qs_slots + threadIdx.x);
  constexpr uint32_t SLOT = QS_THREADS * sizeof(float4);
  float2 f1[QS_BG], f2[QS_BG];
#pragma unroll
  for (int b = 0; b < QS_BG; ++b) { f1[b] = make_float2(0.f, 0.f); f2[b] = f1[b]; }
  unsigned dirt = 0u;            // one bit per band of the group
  int nval = 0;
  long long q = q0 + threadIdx.x;
  bool has = q < q1;
  {
    const char* pb = reinterpret_cast<const char*>(a.cube) + ((long long)g0 * n4 + q) * (long long)sizeof(float4);
#pragma unroll
    for (int b = 0; b < QS_BG; ++b) {
      if (has && (FULL || g0 + b < B)) cp_async16(slot0 + b * SLOT, pb);
      cp_commit();
      pb += sb; pin(pb);
    }
  }
  unsigned wm = has ? __ldg(reinterpret_cast<const unsigned*>(a.W) + q) : 0u;
  while (has) {
    const long long qn = q + QS_THREADS;
    const bool hasn = qn < q1;
    const unsigned wmn = hasn ? __ldg(reinterpret_cast<const unsigned*>(a.W) + qn) : 0u;
    nval += __popc(wm & 0x01010101u);
    const bool edge = (wm & 0x01010101u) != 0x01010101u;          // some invalid pixel in the group
    // per pixel: all ones where valid (keeps the value), 0x7fffffff where invalid (|x| != 0 there = not clean)
    const unsigned k0 = (wm & 0x000000ffu) ? 0xffffffffu : 0u, k1 = (wm & 0x0000ff00u) ? 0xffffffffu : 0u,
                   k2 = (wm & 0x00ff0000u) ? 0xffffffffu : 0u, k3 = (wm & 0xff000000u) ? 0xffffffffu : 0u;
    unsigned kk0 = k0, kk1 = k1, kk2 = k2, kk3 = k3;
    pin(kk0); pin(kk1); pin(kk2); pin(kk3);
    float2 s01 = make_float2(0.f, 0.f), s23 = s01;
    if (g0 > 0 && want_sum) { const float4 sp = reinterpret_cast<const float4*>(a.sum_out)[q]; s01 = make_float2(sp.x, sp.y); s23 = make_float2(sp.z, sp.w); }
    const char* pb = reinterpret_cast<const char*>(a.cube) + ((long long)g0 * n4 + qn) * (long long)sizeof(float4);
#pragma unroll
    for (int b = 0; b < QS_BG; ++b) {
      cp_wait<QS_BG - 1>();
      const bool live = FULL || g0 + b < B;
      const float4 x = live ? qs_slots[b * QS_THREADS + threadIdx.x] : make_float4(0.f, 0.f, 0.f, 0.f);
      const float2 x01 = make_float2(x.x, x.y), x23 = make_float2(x.z, x.w);
      const float np = -s_piv[live ? g0 + b : 0];
      float2 t01 = q_add2(x01, make_float2(np, np)), t23 = q_add2(x23, make_float2(np, np));
      if (edge) {     // invalid pixels count as 0 whatever they hold (NaN and Inf included)
        t01.x = __uint_as_float(__float_as_uint(t01.x) & kk0); t01.y = __uint_as_float(__float_as_uint(t01.y) & kk1);
        t23.x = __uint_as_float(__float_as_uint(t23.x) & kk2); t23.y = __uint_as_float(__float_as_uint(t23.y) & kk3);
        const unsigned dz = ((__float_as_uint(x.x) & ~kk0) | (__float_as_uint(x.y) & ~kk1) | (__float_as_uint(x.z) & ~kk2) |
                             (__float_as_uint(x.w) & ~kk3)) & 0x7fffffffu;
        if (dz) dirt |= 1u << b;
      }
      f1[b] = q_add2(f1[b], q_add2(t01, t23));
      f2[b] = q_fma2(t01, t01, q_fma2(t23, t23, f2[b]));
      s01 = q_add2(s01, x01); s23 = q_add2(s23, x23);
      if (hasn && live) cp_async16(slot0 + b * SLOT, pb);
      cp_commit();
      pb += sb; pin(pb);
    }
    if (want_sum) reinterpret_cast<float4*>(a.sum_out)[q] = make_float4(s01.x, s01.y, s23.x, s23.y);
    q = qn; has = hasn; wm = wmn;
  }
  cp_wait<0>();
  // block reduction: fp32 across the warp (a few hundred values), float64 from there on
#pragma unroll
  for (int b = 0; b < QS_BG; ++b) {
    float v1 = f1[b].x + f1[b].y, v2 = f2[b].x + f2[b].y;
    v1 = lpf_warp_sum(v1); v2 = lpf_warp_sum(v2);
    if (lane == 0) { s_red[warp][b][0] = (double)v1; s_red[warp][b][1] = (double)v2; }
  }
  const unsigned any_dirt = __reduce_or_sync(0xffffffffu, dirt);
  if (any_dirt && lane == 0)
    for (int b = 0; b < QS_BG; ++b)
      if (((any_dirt >> b) & 1u) && g0 + b < B) a.dirty_b[g0 + b] = a.seq;
  nval = lpf_warp_sum(nval);
  if (lane == 0) s_n[warp] = (double)nval;
  __syncthreads();
  if (threadIdx.x < QS_BG && g0 + threadIdx.x < B) {
    double t1 = 0, t2 = 0, tn = 0;
#pragma unroll
    for (int w = 0; w < QS_WARPS; ++w) { t1 += s_red[w][threadIdx.x][0]; t2 += s_red[w][threadIdx.x][1]; tn += s_n[w]; }
    double* o = a.part1 + ((long long)(g0 + threadIdx.x) * gridDim.x + blockIdx.x) * 3;
    o[0] = tn; o[1] = t1; o[2] = t2;
  }
  __syncthreads();
}

__global__ void __launch_bounds__(QS_THREADS, LPF_QS_BLOCKS)
k_qc_moments(const QsArgs a_in) {
  QsArgs a = a_in;
  if (a.fd) { a.cube = a.fd->cube; a.seq = a.fd->seq; }
  extern __shared__ float4 qs_slots[];     // [QS_BG][QS_THREADS]
  __shared__ float s_piv[LPF_MAX_BANDS];
  __shared__ double s_red[QS_WARPS][QS_BG][2];
  __shared__ double s_n[QS_WARPS];
  const int B = a.B;
  const long long N = a.N, n4 = N >> 2;
  for (int b = threadIdx.x; b < B; b += QS_THREADS) s_piv[b] = a.cube[(long long)b * N + a.first_valid];
  __syncthreads();
  const long long per = (n4 + gridDim.x - 1) / gridDim.x;
  const long long q0 = (long long)blockIdx.x * per, q1 = q0 + per < n4 ? q0 + per : n4;
  for (int g0 = 0; g0 < B; g0 += QS_BG) {
    if (g0 + QS_BG <= B) qs_moments_group<true>(a, g0, q0, q1, s_piv, s_red, s_n, qs_slots);
    else qs_moments_group<false>(a, g0, q0, q1, s_piv, s_red, s_n, qs_slots);
  }
}

struct QvArgs {
  QcArgs q;                 // partials [B][nblk][3] and everything the verdict writes
  const int32_t* dirty_b; int seq; int32_t* dirty;   // -> *dirty = seq when an accepted band is not clean outside the mask
  int32_t* zero_me;         // a counter this kernel resets (the record count of the frame), or null
  double* mom;              // [B][3] scratch: the finished sums of every band
};

// sum of three doubles over the block (QC_THREADS threads); valid in thread 0
__device__ __forceinline__ void block_sum3(double& a, double& b, double& c) {
  __shared__ double s_bs[3][QC_WARPS];
  a = lpf_warp_sum(a); b = lpf_warp_sum(b); c = lpf_warp_sum(c);
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  if (l == 0) { s_bs[0][w] = a; s_bs[1][w] = b; s_bs[2][w] = c; }
  __syncthreads();
  if (threadIdx.x == 0) {
    a = 0; b = 0; c = 0;
#pragma unroll
    for (int i = 0; i < QC_WARPS; ++i) { a += s_bs[0][i]; b += s_bs[1][i]; c += s_bs[2][i]; }
  }
}

// one block per band sums that band's partials (one load round); the last block to finish evaluates eq. A.1
__global__ void __launch_bounds__(QC_THREADS)
k_qc_verdict(const QvArgs a_in) {
  QvArgs a = a_in;
  if (a.q.fd) { a.q.cube = a.q.fd->cube; a.seq = a.q.fd->seq; }
  const int b = blockIdx.x, nblk = a.q.nblk;
  double n = 0, s1 = 0, s2 = 0;
  for (int i = threadIdx.x; i < nblk; i += QC_THREADS) {
    const double* q = a.q.part1 + ((long long)b * nblk + i) * 3;
    n += __ldcg(q); s1 += __ldcg(q + 1); s2 += __ldcg(q + 2);
  }
  block_sum3(n, s1, s2);
  if (threadIdx.x == 0) { a.mom[3 * b] = n; a.mom[3 * b + 1] = s1; a.mom[3 * b + 2] = s2; }
  if (!last_block_done(a.q.counter, gridDim.x)) return;
  const int dirt = ((int)threadIdx.x < a.q.B) ? (__ldcg(&a.dirty_b[threadIdx.x]) == a.seq) : 0;   // asked for before the verdict
  qc_verdict(a.q, a.mom);
  const bool mine = (int)threadIdx.x < a.q.B && dirt && a.q.band_ok[threadIdx.x];   // band_ok[t] was written by this thread
  const int bad = __syncthreads_or(mine ? 1 : 0);
  if (threadIdx.x == 0) {
    if (bad) *a.dirty = a.seq;
    if (a.zero_me) *a.zero_me = 0;
  }
}

struct QkArgs {
  const LpfFrameDesc* fd;
  const float* cube; const uint8_t* W; const uint8_t* band_ok; long long N; int B;
  const float* band_clip;  // [B][2]
  double* part2;           // [gridDim.x][B][3]
  float* sum_out;          // [N]: rebuilt from the accepted bands when a band was rejected; or null
};

template <bool FULL, bool RESUM>
__device__ __forceinline__ void qs_clip_group(const QkArgs& a, int g0, long long q0, long long q1, const float* s_c,
                                              const float* s_w, const uint8_t* s_ok, double (*s_red)[QS_BG][3], float4* qs_slots) {
  const int B = a.B, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const long long n4 = a.N >> 2;
  const long long sb = n4 * (long long)sizeof(float4);
  const uint32_t slot0 = (uint32_t)__cvta_generic_to_shared(qs_slots + threadIdx.x);
  constexpr uint32_t SLOT = QS_THREADS * sizeof(float4);
  float fn[QS_BG], f1[QS_BG], f2[QS_BG];     // fn: a count (a thread sees a few dozen pixels: exact in fp32)
#pragma unroll
  for (int b = 0; b < QS_BG; ++b) { fn[b] = 0.f; f1[b] = 0.f; f2[b] = 0.f; }
  long long q = q0 + threadIdx.x;
  bool has = q < q1;
  {
    const char* pb = reinterpret_cast<const char*>(a.cube) + ((long long)g0 * n4 + q) * (long long)sizeof(float4);
#pragma unroll
    for (int b = 0; b < QS_BG; ++b) {
      if (has && (FULL || g0 + b < B)) cp_async16(slot0 + b * SLOT, pb);
      cp_commit();
      pb += sb; pin(pb);
    }
  }
  unsigned wm = has ? __ldg(reinterpret_cast<const unsigned*>(a.W) + q) : 0u;
  while (has) {
    const long long qn = q + QS_THREADS;
    const bool hasn = qn < q1;
    const unsigned wmn = hasn ? __ldg(reinterpret_cast<const unsigned*>(a.W) + qn) : 0u;
    // an invalid pixel never passes: its validity is the second operand of the comparison's predicate
    const bool vk[4] = {(wm & 0x000000ffu) != 0u, (wm & 0x0000ff00u) != 0u, (wm & 0x00ff0000u) != 0u, (wm & 0xff000000u) != 0u};
    float4 sp = make_float4(0.f, 0.f, 0.f, 0.f);
    if (RESUM && g0 > 0) sp = reinterpret_cast<const float4*>(a.sum_out)[q];
    const char* pb = reinterpret_cast<const char*>(a.cube) + ((long long)g0 * n4 + qn) * (long long)sizeof(float4);
#pragma unroll
    for (int b = 0; b < QS_BG; ++b) {
      cp_wait<QS_BG - 1>();
      const bool live = FULL || g0 + b < B;
      const int bb = live ? g0 + b : 0;
      const float4 x = live ? qs_slots[b * QS_THREADS + threadIdx.x] : make_float4(0.f, 0.f, 0.f, 0.f);
      const float c = s_c[bb], w = live ? s_w[bb] : -1.f;
      const float xv[4] = {x.x, x.y, x.z, x.w};
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const float d = xv[j] - c;
        if (fabsf(d) <= w && vk[j]) { fn[b] += 1.f; f1[b] += d; f2[b] = fmaf(d, d, f2[b]); }   // three predicated instructions
      }
      if (RESUM && live && s_ok[bb]) { sp.x += x.x; sp.y += x.y; sp.z += x.z; sp.w += x.w; }
      if (hasn && live) cp_async16(slot0 + b * SLOT, pb);
      cp_commit();
      pb += sb; pin(pb);
    }
    if (RESUM) reinterpret_cast<float4*>(a.sum_out)[q] = sp;
    q = qn; has = hasn; wm = wmn;
  }
  cp_wait<0>();
#pragma unroll
  for (int b = 0; b < QS_BG; ++b) {
    const float vn = lpf_warp_sum(fn[b]), v1 = lpf_warp_sum(f1[b]), v2 = lpf_warp_sum(f2[b]);
    if (lane == 0) { s_red[warp][b][0] = (double)vn; s_red[warp][b][1] = (double)v1; s_red[warp][b][2] = (double)v2; }
  }
  __syncthreads();
  if (threadIdx.x < QS_BG && g0 + threadIdx.x < B) {
    double t0 = 0, t1 = 0, t2 = 0;
#pragma unroll
    for (int w = 0; w < QS_WARPS; ++w) { t0 += s_red[w][threadIdx.x][0]; t1 += s_red[w][threadIdx.x][1]; t2 += s_red[w][threadIdx.x][2]; }
    double* o = a.part2 + ((long long)blockIdx.x * B + g0 + threadIdx.x) * 3;
    o[0] = t0; o[1] = t1; o[2] = t2;
  }
  __syncthreads();
}

__global__ void __launch_bounds__(QS_THREADS, LPF_QS_BLOCKS)
k_qc_clip(const QkArgs a_in) {
  QkArgs a = a_in;
  if (a.fd) a.cube = a.fd->cube;
  extern __shared__ float4 qs_slots[];     // [QS_BG][QS_THREADS]
  __shared__ float s_c[LPF_MAX_BANDS], s_w[LPF_MAX_BANDS];
  __shared__ uint8_t s_ok[LPF_MAX_BANDS + 1];
  __shared__ double s_red[QS_WARPS][QS_BG][3];
  __shared__ int s_rej;
  const int B = a.B;
  const long long n4 = a.N >> 2;
  if (threadIdx.x == 0) s_rej = 0;
  __syncthreads();
  for (int b = threadIdx.x; b <= B; b += QS_THREADS) {
    s_ok[b] = a.band_ok[b];
    if (b < B) { s_c[b] = a.band_clip[2 * b]; s_w[b] = a.band_clip[2 * b + 1]; if (!s_ok[b]) s_rej = 1; }
  }
  __syncthreads();
  const bool resum = a.sum_out != nullptr && s_rej != 0 && s_ok[B] != 0;   // a rejected frame has no sum plane
  const long long per = (n4 + gridDim.x - 1) / gridDim.x;
  const long long q0 = (long long)blockIdx.x * per, q1 = q0 + per < n4 ? q0 + per : n4;
  for (int g0 = 0; g0 < B; g0 += QS_BG) {
    const bool full = g0 + QS_BG <= B;
    if (full && !resum) qs_clip_group<true, false>(a, g0, q0, q1, s_c, s_w, s_ok, s_red, qs_slots);
    else if (full) qs_clip_group<true, true>(a, g0, q0, q1, s_c, s_w, s_ok, s_red, qs_slots);
    else if (!resum) qs_clip_group<false, false>(a, g0, q0, q1, s_c, s_w, s_ok, s_red, qs_slots);
    else qs_clip_group<false, true>(a, g0, q0, q1, s_c, s_w, s_ok, s_red, qs_slots);
  }
}

// one block per band: the clipped mean / rms from the per-block partials [nblk][B][3]
__global__ void __launch_bounds__(QC_THREADS)
k_qc_clip_finish(const double* part2, int nblk, int B, const float* band_clip, float* stats) {
  const int b = blockIdx.x;
  double nc = 0, c1 = 0, c2 = 0;
  for (int i = threadIdx.x; i < nblk; i += QC_THREADS) {
    const double* r = part2 + ((long long)i * B + b) * 3;
    nc += __ldcg(r); c1 += __ldcg(r + 1); c2 += __ldcg(r + 2);
  }
  block_sum3(nc, c1, c2);
  if (threadIdx.x == 0) {
    double cmean = 0, crms = 0;
    if (nc > 0) {
      const double k1 = c1 / nc;
      cmean = (double)band_clip[2 * b] + k1;         // the clip pass is centred on the fp32 mean
      const double cv = c2 / nc - k1 * k1;
      crms = sqrt(cv > 0 ? cv : 0.0);
    }
    float* o = stats + LPF_STATS_PER_BAND * b;
    o[3] = (float)nc; o[4] = (float)cmean; o[5] = (float)crms;
  }
}

// ---- O12: per-pixel running quality control (eq. A.2; R22) -------------------
// One block per (chunk, band).  zeta = (x - mean) / sqrt(var) is tested as d*d > thr^2 * var at valid pixels with
// var > 0; the Welford / exponentially weighted update of the frame is written to the OTHER copy of the state and
// adopted per band by the last block, which also folds the verdict into band_ok / frame_ok ("test before update,
// update only accepted bands") and applies the start-over rule (zeta_reset consecutive discards).
struct RqArgs {
  const float* cube; const uint8_t* W; long long N; int B, nblk;
  float* m; float* v;            // [2][B][N]
  int32_t* cur; int32_t* nupd; int32_t* cnt; int32_t* run; int32_t* counter;   // [B], [B], [B], [B], [1]
  float thr2; int nmax, window, warm, reset;
  uint8_t* band_ok; int32_t* zeta_cnt;
};

__device__ __forceinline__ void rq_pixel(float x, float m, float v, bool test, float a, float one_m_a, float thr2,
                                         float& m2, float& v2, int& hits) {
  const float d = x - m;
  if (test && v > 0.f && d * d > thr2 * v) ++hits;
  m2 = fmaf(a, d, m);
  v2 = one_m_a * fmaf(a * d, d, v);
}

__global__ void __launch_bounds__(QC_THREADS)
k_qc_running(const RqArgs a) {
  __shared__ int s_hits[QC_WARPS];
  const int b = blockIdx.y, nblk = a.nblk;
  const long long N = a.N;
  const int cur = a.cur[b], nup = a.nupd[b];
  const bool tested = nup >= a.warm;
  const int k = nup + 1 < a.window ? nup + 1 : a.window;
  const float al = 1.0f / (float)k, oma = 1.0f - al;
  const bool fresh = nup == 0;       // a band that starts (over): its state counts as zero
  const float* X = a.cube + (long long)b * N;
  const float* m0 = a.m + ((long long)cur * a.B + b) * N;
  const float* v0 = a.v + ((long long)cur * a.B + b) * N;
  float* m1 = a.m + ((long long)(cur ^ 1) * a.B + b) * N;
  float* v1 = a.v + ((long long)(cur ^ 1) * a.B + b) * N;
  const long long n4 = (N + 3) >> 2;
  const long long per = (n4 + nblk - 1) / nblk;
  const long long q0 = (long long)blockIdx.x * per;
  const long long q1 = (q0 + per < n4) ? q0 + per : n4;
  const bool vec = ((N & 3) == 0) && ((((uintptr_t)a.cube) & 15) == 0);
  int hits = 0;
  if (vec) {
    for (long long q = q0 + threadIdx.x; q < q1; q += QC_THREADS) {
      const float4 x = __ldg(reinterpret_cast<const float4*>(X) + q);
      float4 m = *(reinterpret_cast<const float4*>(m0) + q), v = *(reinterpret_cast<const float4*>(v0) + q);
      if (fresh) { m = make_float4(0.f, 0.f, 0.f, 0.f); v = m; }
      const unsigned wm = __ldg(reinterpret_cast<const unsigned*>(a.W) + q);
      float4 m2, v2;
      rq_pixel(x.x, m.x, v.x, tested && (wm & 0x000000ffu), al, oma, a.thr2, m2.x, v2.x, hits);
      rq_pixel(x.y, m.y, v.y, tested && (wm & 0x0000ff00u), al, oma, a.thr2, m2.y, v2.y, hits);
      rq_pixel(x.z, m.z, v.z, tested && (wm & 0x00ff0000u), al, oma, a.thr2, m2.z, v2.z, hits);
      rq_pixel(x.w, m.w, v.w, tested && (wm & 0xff000000u), al, oma, a.thr2, m2.w, v2.w, hits);
      *(reinterpret_cast<float4*>(m1) + q) = m2; *(reinterpret_cast<float4*>(v1) + q) = v2;
    }
  } else {
    for (long long i = (q0 << 2) + threadIdx.x; i < (q1 << 2) && i < N; i += QC_THREADS) {
      float m2, v2;
      rq_pixel(X[i], fresh ? 0.f : m0[i], fresh ? 0.f : v0[i], tested && a.W[i] != 0, al, oma, a.thr2, m2, v2, hits);
      m1[i] = m2; v1[i] = v2;
    }
  }
  hits = lpf_warp_sum(hits);
  if ((threadIdx.x & 31) == 0) s_hits[threadIdx.x >> 5] = hits;
  __syncthreads();
  if (threadIdx.x == 0) {
    int t = 0;
    for (int w = 0; w < QC_WARPS; ++w) t += s_hits[w];
    if (t) atomicAdd(&a.cnt[b], t);
  }
  if (!last_block_done(a.counter, gridDim.x * gridDim.y)) return;
  __shared__ int s_nok;
  if (threadIdx.x == 0) s_nok = 0;
  __syncthreads();
  if (threadIdx.x < a.B) {
    const int bb = threadIdx.x;
    const int c = __ldcg(&a.cnt[bb]);
    const int nu = a.nupd[bb];
    const int ok_in = a.band_ok[bb];
    const bool discard = nu >= a.warm && c > a.nmax;          // eq. A.2
    const int ok = (ok_in && !discard) ? 1 : 0;
    if (ok) { a.cur[bb] ^= 1; a.nupd[bb] = nu + 1; a.run[bb] = 0; atomicAdd(&s_nok, 1); }
    else if (ok_in && discard) {
      const int r = a.run[bb] + 1;
      if (a.reset > 0 && r >= a.reset) { a.nupd[bb] = 0; a.run[bb] = 0; }   // the band starts over
      else a.run[bb] = r;
    }
    a.band_ok[bb] = (uint8_t)ok;
    a.zeta_cnt[bb] = c;
    a.cnt[bb] = 0;
  }
  __syncthreads();
  if (threadIdx.x == 0) a.band_ok[a.B] = (s_nok >= (a.B + 1) / 2) ? 1 : 0;
}

}  // namespace

static Qc2Args make_qc2(lpf_ctx* c, LpfLane& L, const float* d_cube, const uint8_t* d_band_ok, float* d_stats, bool want_sum,
                        int32_t* zero_me) {
  Qc2Args a{};
  a.cube = d_cube; a.W = c->W; a.band_ok = d_band_ok; a.N = c->N; a.B = c->p.B;
  a.band_clip = L.qc_band_clip; a.part2 = L.qc_part2; a.stats = d_stats;
  a.sum_out = want_sum ? L.sum_plane : nullptr;
  a.dirty = L.dirty; a.seq = L.dirty_seq; a.zero_me = zero_me; a.counter = L.qc_counter + 1;
  return a;
}

static int qc_launch_pass1(lpf_ctx* c, LpfLane& L, const float* d_cube, float* d_stats, uint8_t* d_band_ok, cudaStream_t st) {
  QcArgs a{};
  a.cube = d_cube; a.W = c->W; a.N = c->N; a.first_valid = c->first_valid; a.B = c->p.B; a.nblk = c->qc_nblk;
  a.part1 = L.qc_part1; a.qc_clip = c->p.qc_clip; a.tau = c->p.qc_tau; a.stats = d_stats; a.band_ok = d_band_ok;
  a.band_clip = L.qc_band_clip; a.counter = L.qc_counter; a.big_thr = L.big_thr; a.big_sigma = lpf_fused_big_sigma();
  const dim3 grid(c->qc_nblk, c->p.B);
  LPF_KLAUNCH(c, KID_QC_PASS1, st, k_qc_pass1<<<grid, QC_THREADS, 0, st>>>(a));
  return LPF_OK;
}

int lpf_qc2_blocks(const lpf_ctx* c) {
  const long long chunks = ((c->N + 3) / 4 + 4 * QC2_THREADS - 1) / (4 * QC2_THREADS);
  const long long cap = (long long)c->n_sm * 8;
  return (int)(chunks < 1 ? 1 : (chunks < cap ? chunks : cap));
}

// O12 between the two passes (when zeta_thr > 0).  The state is one recurrence over the frames, so the calls of
// different lanes are ordered by an event.
int lpf_launch_qc_running(lpf_ctx* c, LpfLane& L, const float* d_cube, uint8_t* d_band_ok, cudaStream_t st) {
  const lpf_params& p = c->p;
  if (!(p.zeta_thr > 0)) return LPF_OK;
  if (c->rq_valid) LPF_CUDA(cudaStreamWaitEvent(st, c->rq_ev, 0));
  RqArgs a{};
  a.cube = d_cube; a.W = c->W; a.N = c->N; a.B = p.B; a.nblk = c->qc_nblk;
  a.m = c->rq_m; a.v = c->rq_v; a.cur = c->rq_state; a.nupd = c->rq_state + p.B; a.cnt = c->rq_state + 2 * p.B;
  a.run = c->rq_state + 3 * p.B; a.counter = c->rq_state + 4 * p.B;
  a.thr2 = p.zeta_thr * p.zeta_thr; a.nmax = p.zeta_nmax; a.window = p.zeta_window; a.warm = p.zeta_warm; a.reset = p.zeta_reset;
  a.band_ok = d_band_ok; a.zeta_cnt = L.zeta_cnt;
  const dim3 grid(c->qc_nblk, p.B);
  LPF_KLAUNCH(c, KID_QC_VERDICT, st, k_qc_running<<<grid, QC_THREADS, 0, st>>>(a));
  LPF_CUDA(cudaEventRecord(c->rq_ev, st));
  c->rq_valid = true;
  return LPF_OK;
}

// Grid of the streaming kernels: blocks of about 28 (pixel group, band group) rounds per thread - long enough to
// amortise a block's start and its reductions, short enough to balance - twice as many when fewer than 4 lanes are in
// flight (a kernel alone on the GPU wants more bytes in flight); between one wave of single blocks and the 5 blocks
// per SM the registers allow.  Measured on configs 3, 4, 5.
int lpf_qs_blocks(const lpf_ctx* c) {
  const long long n4 = (c->N + 3) / 4, nbg = (c->p.B + QS_BG - 1) / QS_BG;
  const long long want = (n4 + QS_THREADS - 1) / QS_THREADS;
  long long nb = (n4 * nbg + 28ll * QS_THREADS - 1) / (28ll * QS_THREADS);
  if (c->p.n_lanes < 4) nb *= 2;
  const long long lo = want < c->n_sm ? want : c->n_sm, hi = (long long)LPF_QS_BLOCKS * c->n_sm;
  nb = nb < lo ? lo : (nb > hi ? hi : nb);
  nb = nb > want ? want : nb;
  return (int)(nb < 1 ? 1 : nb);
}

// the dynamic shared memory attribute, once per process (16 KB needs no opt-in; a larger LPF_QS_* build does)
static cudaError_t qs_attr() {
  static bool done = false;
  if (done) return cudaSuccess;
  cudaError_t e = cudaFuncSetAttribute(k_qc_moments, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)QS_SMEM);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_qc_clip, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)QS_SMEM);
  done = e == cudaSuccess;
  return e;
}

// the kernel attributes, once per process, outside any stream capture (lpf_create)
int lpf_qc_prepare(void) {
  LPF_CUDA(qs_attr());
  return LPF_OK;
}

// the streaming form needs 128-bit loads of every band at the same pixel group
static bool qc_streaming(const lpf_ctx* c, const float* d_cube) { return (c->N & 3) == 0 && (((uintptr_t)d_cube) & 15) == 0; }

// moments + verdict (+ speculative sum plane, + reset of *zero_me), streaming form
static int qs_launch_moments(lpf_ctx* c, LpfLane& L, const float* d_cube, float* d_stats, uint8_t* d_band_ok, bool want_sum,
                             int32_t* zero_me, cudaStream_t st) {
  const int nblk = lpf_qs_blocks(c);
  L.dirty_seq = L.dirty_seq >= 0x7ffffff0 ? 1 : L.dirty_seq + 1;
  QsArgs m{};
  m.fd = c->cap_fd; m.cube = d_cube; m.W = c->W; m.N = c->N; m.first_valid = c->first_valid; m.B = c->p.B; m.part1 = L.qc_part1;
  m.sum_out = want_sum ? L.sum_plane : nullptr; m.dirty_b = L.dirty_b; m.seq = L.dirty_seq;
  LPF_CUDA(qs_attr());
  LPF_KLAUNCH(c, KID_QC_PASS1, st, k_qc_moments<<<nblk, QS_THREADS, QS_SMEM, st>>>(m));
  QvArgs v{};
  v.q.fd = c->cap_fd; v.q.cube = d_cube; v.q.W = c->W; v.q.N = c->N; v.q.first_valid = c->first_valid; v.q.B = c->p.B; v.q.nblk = nblk;
  v.q.part1 = L.qc_part1; v.q.qc_clip = c->p.qc_clip; v.q.tau = c->p.qc_tau; v.q.stats = d_stats; v.q.band_ok = d_band_ok;
  v.q.band_clip = L.qc_band_clip; v.q.counter = L.qc_counter; v.q.big_thr = L.big_thr; v.q.big_sigma = lpf_fused_big_sigma();
  v.dirty_b = L.dirty_b; v.seq = L.dirty_seq; v.dirty = L.dirty; v.zero_me = zero_me; v.mom = L.qc_mom;
  LPF_KLAUNCH(c, KID_QC_VERDICT1, st, k_qc_verdict<<<c->p.B, QC_THREADS, 0, st>>>(v));
  return LPF_OK;
}

static int qs_launch_clip(lpf_ctx* c, LpfLane& L, const float* d_cube, float* d_stats, const uint8_t* d_band_ok, bool want_sum,
                          cudaStream_t st) {
  const int nblk = lpf_qs_blocks(c);
  QkArgs k{};
  k.fd = c->cap_fd; k.cube = d_cube; k.W = c->W; k.band_ok = d_band_ok; k.N = c->N; k.B = c->p.B; k.band_clip = L.qc_band_clip; k.part2 = L.qc_part2;
  k.sum_out = want_sum ? L.sum_plane : nullptr;
  LPF_CUDA(qs_attr());
  LPF_KLAUNCH(c, KID_QC_PASS2, st, k_qc_clip<<<nblk, QS_THREADS, QS_SMEM, st>>>(k));
  LPF_KLAUNCH(c, KID_QC_CLIPFIN, st, k_qc_clip_finish<<<c->p.B, QC_THREADS, 0, st>>>(L.qc_part2, nblk, c->p.B, L.qc_band_clip, d_stats));
  return LPF_OK;
}

// S1 + S2 as the C-ABI's lpf_cube_qc: statistics and verdict only.
int lpf_launch_qc(lpf_ctx* c, LpfLane& L, const float* d_cube, float* d_stats, uint8_t* d_band_ok, cudaStream_t st) {
  if (qc_streaming(c, d_cube)) {
    int rc = qs_launch_moments(c, L, d_cube, d_stats, d_band_ok, false, nullptr, st);
    if (rc) return rc;
    rc = lpf_launch_qc_running(c, L, d_cube, d_band_ok, st);
    if (rc) return rc;
    return qs_launch_clip(c, L, d_cube, d_stats, d_band_ok, false, st);
  }
  int rc = qc_launch_pass1(c, L, d_cube, d_stats, d_band_ok, st);
  if (rc) return rc;
  rc = lpf_launch_qc_running(c, L, d_cube, d_band_ok, st);
  if (rc) return rc;
  const Qc2Args a = make_qc2(c, L, d_cube, d_band_ok, d_stats, false, nullptr);
  LPF_KLAUNCH(c, KID_QC_PASS2, st, k_qc_pass2<true, false><<<lpf_qc2_blocks(c), QC2_THREADS, 0, st>>>(a));
  return LPF_OK;
}

// S1 + S2 + S3 for the chained frame call; *zero_me (the frame's record counter) is reset on the way.
// Streaming form: the sum plane comes out of the first read of the cube (all bands; the clip pass rebuilds it
// when the verdict rejected a band).  Generic form: the clip round, the sum plane and the exact-zero check share
// the second read.
int lpf_launch_qc_sum(lpf_ctx* c, LpfLane& L, const float* d_cube, float* d_stats, uint8_t* d_band_ok, int32_t* zero_me,
                      cudaStream_t st) {
  const bool want_sum = c->p.detect_sum_plane != 0;
  if (qc_streaming(c, d_cube)) {
    int rc = qs_launch_moments(c, L, d_cube, d_stats, d_band_ok, want_sum, zero_me, st);
    if (rc) return rc;
    rc = lpf_launch_qc_running(c, L, d_cube, d_band_ok, st);
    if (rc) return rc;
    return qs_launch_clip(c, L, d_cube, d_stats, d_band_ok, want_sum, st);
  }
  int rc = qc_launch_pass1(c, L, d_cube, d_stats, d_band_ok, st);
  if (rc) return rc;
  rc = lpf_launch_qc_running(c, L, d_cube, d_band_ok, st);
  if (rc) return rc;
  L.dirty_seq = L.dirty_seq >= 0x7ffffff0 ? 1 : L.dirty_seq + 1;
  const Qc2Args a = make_qc2(c, L, d_cube, d_band_ok, d_stats, want_sum, zero_me);
  LPF_KLAUNCH(c, KID_QC_PASS2, st, k_qc_pass2<true, true><<<lpf_qc2_blocks(c), QC2_THREADS, 0, st>>>(a));
  return LPF_OK;
}

// S3 alone (lpf_detect_sources): the sum plane of the accepted bands (want_sum) and the exact-zero check.
int lpf_launch_sum_plane(lpf_ctx* c, LpfLane& L, const float* d_cube, const uint8_t* d_band_ok, bool want_sum, cudaStream_t st) {
  L.dirty_seq = L.dirty_seq >= 0x7ffffff0 ? 1 : L.dirty_seq + 1;
  const Qc2Args a = make_qc2(c, L, d_cube, d_band_ok, nullptr, want_sum, nullptr);
  LPF_KLAUNCH(c, KID_SUM_PLANE, st, k_qc_pass2<false, true><<<lpf_qc2_blocks(c), QC2_THREADS, 0, st>>>(a));
  return LPF_OK;
}

// ---- lpf_cube_qc_static: S1 + S2 with no allocation behind it -------------------------------------------------------
// For callers that must not (or cannot) reach cudaMalloc: the per-block partial sums, the clip parameters, the noise
// levels and the two block counters of the generic QC kernels live in ONE file-scope device array instead of a
// lane's buffers.  Every GPU that loads the library holds LPF_QC_STATIC_BYTES of it until the process exits; every
// call on a device shares it (calls that overlap on the GPU race) and finds the last call's contents in it (the
// counters, which must start at zero, are cleared on the stream first; everything else is written before it is read).
// In host code the array's name is a host-side stand-in, not a device address: the kernels get the address that
// cudaGetSymbolAddress returns for the current device, asked for once per device.
static __device__ __align__(256) unsigned char g_qc_static[LPF_QC_STATIC_BYTES];

namespace {
constexpr size_t QST_COUNTERS = 0;                                       // 2 x int32
constexpr size_t QST_BAND_CLIP = 256;                                    // [LPF_MAX_BANDS][2] float
constexpr size_t QST_BIG_THR = 1024;                                     // [LPF_MAX_BANDS + 1] float
constexpr size_t QST_PART = 2048;                                        // part1 [B][nblk1][3], then part2 [nblk2][B][3], double
constexpr int QST_MAX_DEV = 64;
static_assert(QST_BAND_CLIP + LPF_MAX_BANDS * 2 * sizeof(float) <= QST_BIG_THR, "static QC scratch layout");
static_assert(QST_BIG_THR + (LPF_MAX_BANDS + 1) * sizeof(float) <= QST_PART, "static QC scratch layout");

// device address of g_qc_static on the current device (set-up: the first call on that device)
int qc_static_base(unsigned char** out) {
  static unsigned char* base[QST_MAX_DEV] = {};
  int dev = -1;
  LPF_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= QST_MAX_DEV) return LPF_E_ARG;
  if (!base[dev]) {
    unsigned char* p = nullptr;
    LPF_CUDA(cudaGetSymbolAddress((void**)&p, g_qc_static));
    base[dev] = p;
  }
  *out = base[dev];
  return LPF_OK;
}
}  // namespace

extern "C" int lpf_cube_qc_static(lpf_ctx* c, const float* d_cube, float* d_stats, uint8_t* d_band_ok, void* stream) {
  if (!c || !d_cube || !d_stats || !d_band_ok) return LPF_E_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  const int B = c->p.B, nblk1 = c->qc_nblk, nblk2 = lpf_qc2_blocks(c);
  const size_t b1 = (size_t)B * nblk1 * 3 * sizeof(double), b2 = (size_t)nblk2 * B * 3 * sizeof(double);
  const size_t o1 = QST_PART, o2 = (o1 + b1 + 255) & ~(size_t)255, need = o2 + b2;
  if (need > (size_t)LPF_QC_STATIC_BYTES) {
    snprintf(g_lpf_cuda_err, sizeof(g_lpf_cuda_err),
             "lpf_cube_qc_static: B = %d bands x (%d + %d) blocks need %zu bytes of scratch, the static array holds %d "
             "(LPF_QC_STATIC_BYTES); use lpf_cube_qc", B, nblk1, nblk2, need, (int)LPF_QC_STATIC_BYTES);
    return LPF_E_TOO_LARGE;
  }
  unsigned char* base = nullptr;
  int rc = qc_static_base(&base);
  if (rc) return rc;
  int32_t* counters = reinterpret_cast<int32_t*>(base + QST_COUNTERS);
  LPF_CUDA(cudaMemsetAsync(counters, 0, 2 * sizeof(int32_t), st));     // a call that was cut short may have left them set
  QcArgs a{};
  a.cube = d_cube; a.W = c->W; a.N = c->N; a.first_valid = c->first_valid; a.B = B; a.nblk = nblk1;
  a.part1 = reinterpret_cast<double*>(base + o1); a.qc_clip = c->p.qc_clip; a.tau = c->p.qc_tau; a.stats = d_stats; a.band_ok = d_band_ok;
  a.band_clip = reinterpret_cast<float*>(base + QST_BAND_CLIP); a.counter = counters;
  a.big_thr = reinterpret_cast<float*>(base + QST_BIG_THR); a.big_sigma = lpf_fused_big_sigma();
  LPF_KLAUNCH(c, KID_QC_PASS1, st, k_qc_pass1<<<dim3(nblk1, B), QC_THREADS, 0, st>>>(a));
  Qc2Args k{};
  k.cube = d_cube; k.W = c->W; k.band_ok = d_band_ok; k.N = c->N; k.B = B;
  k.band_clip = a.band_clip; k.part2 = reinterpret_cast<double*>(base + o2); k.stats = d_stats;
  k.sum_out = nullptr; k.dirty = nullptr; k.seq = 0; k.zero_me = nullptr; k.counter = counters + 1;
  LPF_KLAUNCH(c, KID_QC_PASS2, st, k_qc_pass2<true, false><<<nblk2, QC2_THREADS, 0, st>>>(k));
  return LPF_OK;
}
