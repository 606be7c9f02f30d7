// S1 + S2: quality control (App. A, eq. A.1; O1, O2).
//
// Pass 1 streams the cube once with 128-bit loads and accumulates, per band over valid
// pixels, n, sum(x - p) and sum(x - p)^2 about a per-band pivot p (the band's first valid
// pixel): fp32 over runs of <= 16 values, float64 across runs, warp-shuffle + shared-memory
// block reduction, one partial per block.  Pass 2 (the cube is L2-resident by then) does the
// same for the pixels inside the one qc_clip-sigma clip round, about the band mean.  The
// verdict kernel finishes the moments and evaluates eq. A.1 across bands (median, MAD, SE
// floor) for the mean vector and the rms vector.
#include "lpf_internal.cuh"

namespace {

constexpr int QC_THREADS = 256;

__device__ __forceinline__ void block_reduce3(double& a, double& b, double& c, double* sm /*[3][8]*/) {
  a = lpf_warp_sum(a); b = lpf_warp_sum(b); c = lpf_warp_sum(c);
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  __syncthreads();
  if (l == 0) { sm[w] = a; sm[8 + w] = b; sm[16 + w] = c; }
  __syncthreads();
  if (w == 0) {
    a = l < (QC_THREADS / 32) ? sm[l] : 0.0;
    b = l < (QC_THREADS / 32) ? sm[8 + l] : 0.0;
    c = l < (QC_THREADS / 32) ? sm[16 + l] : 0.0;
    a = lpf_warp_sum(a); b = lpf_warp_sum(b); c = lpf_warp_sum(c);
  }
}

// CLIP = false: all valid pixels, about pivot.  CLIP = true: |x - mean| <= thr, about mean.
template <bool CLIP>
__global__ void __launch_bounds__(QC_THREADS)
k_qc_moments(const float* __restrict__ cube, const uint8_t* __restrict__ W, long long N, int first_valid,
             int nblk, const double* __restrict__ part1, float qc_clip, double* __restrict__ part_out) {
  __shared__ double sm[24];
  __shared__ float s_piv, s_thr;
  const int b = blockIdx.y;
  const float* X = cube + (long long)b * N;
  if (!CLIP) {
    if (threadIdx.x == 0) { s_piv = X[first_valid]; s_thr = 0.f; }
  } else {
    // finish pass 1 for this band: mean and rms (every block redoes this tiny reduction)
    double n = 0, s1 = 0, s2 = 0;
    for (int i = threadIdx.x; i < nblk; i += QC_THREADS) {
      const double* q = part1 + ((long long)b * nblk + i) * 3;
      n += q[0]; s1 += q[1]; s2 += q[2];
    }
    block_reduce3(n, s1, s2, sm);
    if (threadIdx.x == 0) {
      const double piv = (double)X[first_valid];
      double mean = 0, rms = 0;
      if (n > 0) { const double m1 = s1 / n; mean = piv + m1; double var = s2 / n - m1 * m1; rms = sqrt(var > 0 ? var : 0.0); }
      s_piv = (float)mean;
      s_thr = (float)((double)qc_clip * rms);
    }
  }
  __syncthreads();
  const float piv = s_piv, thr = s_thr;

  // contiguous chunk of this band for this block, in units of 4 pixels
  const long long n4 = (N + 3) >> 2;
  const long long per = (n4 + nblk - 1) / nblk;
  const long long q0 = (long long)blockIdx.x * per;
  const long long q1 = (q0 + per < n4) ? q0 + per : n4;
  const bool vec = ((N & 3) == 0) && ((((uintptr_t)cube) & 15) == 0);

  double dn = 0, d1 = 0, d2 = 0;
  float fn = 0, f1 = 0, f2 = 0;
  int run = 0;
  for (long long q = q0 + threadIdx.x; q < q1; q += QC_THREADS) {
    float v[4]; unsigned wm;
    const long long i0 = q << 2;
    if (vec) {
      const float4 x = __ldg(reinterpret_cast<const float4*>(X) + q);
      v[0] = x.x; v[1] = x.y; v[2] = x.z; v[3] = x.w;
      wm = __ldg(reinterpret_cast<const unsigned*>(W) + q);
    } else {
      wm = 0;
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const bool in = (i0 + j) < N;
        v[j] = in ? X[i0 + j] : 0.f;
        if (in && W[i0 + j]) wm |= (1u << (8 * j));
      }
    }
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const float d = v[j] - piv;
      bool take = ((wm >> (8 * j)) & 0xffu) != 0;
      if (CLIP) take = take && (fabsf(d) <= thr);
      if (take) { fn += 1.f; f1 += d; f2 = fmaf(d, d, f2); }
    }
    if (++run == 4) { dn += fn; d1 += f1; d2 += f2; fn = f1 = f2 = 0.f; run = 0; }
  }
  dn += fn; d1 += f1; d2 += f2;
  block_reduce3(dn, d1, d2, sm);
  if (threadIdx.x == 0) {
    double* o = part_out + ((long long)b * nblk + blockIdx.x) * 3;
    o[0] = dn; o[1] = d1; o[2] = d2;
  }
}

// One block of 64 threads: thread b owns band b.
__global__ void __launch_bounds__(64)
k_qc_verdict(const float* __restrict__ cube, long long N, int first_valid, int B, int nblk,
             const double* __restrict__ part1, const double* __restrict__ part2, float tau,
             float* __restrict__ stats, uint8_t* __restrict__ band_ok) {
  __shared__ double s_mean[64], s_rms[64], s_sorted[64], s_dev[64];
  __shared__ int s_fin[64];
  __shared__ int s_nfin, s_nok;
  const int b = threadIdx.x;
  double n = 0, mean = 0, rms = 0, nc = 0, cmean = 0, crms = 0;
  int fin = 0;
  if (b < B) {
    double s1 = 0, s2 = 0, c1 = 0, c2 = 0;
    for (int i = 0; i < nblk; ++i) {
      const double* q = part1 + ((long long)b * nblk + i) * 3;
      n += q[0]; s1 += q[1]; s2 += q[2];
      const double* r = part2 + ((long long)b * nblk + i) * 3;
      nc += r[0]; c1 += r[1]; c2 += r[2];
    }
    if (n > 0) {
      const double piv = (double)cube[(long long)b * N + first_valid];
      const double m1 = s1 / n;
      mean = piv + m1;
      const double var = s2 / n - m1 * m1;
      rms = sqrt(var > 0 ? var : 0.0);
      if (nc > 0) {
        const double meanf = (double)(float)mean;  // pass 2 centred on the fp32 mean
        const double k1 = c1 / nc;
        cmean = meanf + k1;
        const double cv = c2 / nc - k1 * k1;
        crms = sqrt(cv > 0 ? cv : 0.0);
      }
    }
    fin = (n > 0 && isfinite(mean) && isfinite(rms)) ? 1 : 0;
    s_mean[b] = mean; s_rms[b] = rms; s_fin[b] = fin;
  }
  if (threadIdx.x == 0) { s_nfin = 0; s_nok = 0; }
  __syncthreads();
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
    ok = (fabs(zm) <= (double)tau && fabs(zr) <= (double)tau) ? 1 : 0;
    if (ok) atomicAdd(&s_nok, 1);
  }
  __syncthreads();
  if (b < B) {
    float* o = stats + LPF_STATS_PER_BAND * b;
    o[0] = (float)n; o[1] = (float)mean; o[2] = (float)rms; o[3] = (float)nc; o[4] = (float)cmean; o[5] = (float)crms;
    o[6] = (float)zm; o[7] = (float)zr;
    band_ok[b] = (uint8_t)ok;
  }
  if (threadIdx.x == 0) band_ok[B] = (s_nok >= (B + 1) / 2) ? 1 : 0;
}

}  // namespace

int lpf_launch_qc(lpf_ctx* c, LpfLane& L, const float* d_cube, float* d_stats, uint8_t* d_band_ok, cudaStream_t st) {
  const dim3 grid(c->qc_nblk, c->p.B);
  LPF_KLAUNCH(c, KID_QC_PASS1, st, k_qc_moments<false><<<grid, QC_THREADS, 0, st>>>(
      d_cube, c->W, c->N, c->first_valid, c->qc_nblk, nullptr, 0.f, L.qc_part1));
  LPF_KLAUNCH(c, KID_QC_PASS2, st, k_qc_moments<true><<<grid, QC_THREADS, 0, st>>>(
      d_cube, c->W, c->N, c->first_valid, c->qc_nblk, L.qc_part1, c->p.qc_clip, L.qc_part2));
  LPF_KLAUNCH(c, KID_QC_VERDICT, st, k_qc_verdict<<<1, 64, 0, st>>>(
      d_cube, c->N, c->first_valid, c->p.B, c->qc_nblk, L.qc_part1, L.qc_part2, c->p.qc_tau, d_stats, d_band_ok));
  return LPF_OK;
}
