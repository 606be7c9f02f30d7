// S3-S8, general path: any kernel (Gaussian eq. 2 or box), any n_iter, masks and borders.
// (eqs. 2-7; O3-O6.)
//
// One tiled, register-blocked separable normalised-convolution kernel serves the matched
// filter (F = g_mf (*)_W X), the local centre (C = G (*)_W' F), the local spread
// (S = G (*)_W' (F-C)^2) and, for iterations > 1, the denominators of W' = W and not Y.
// A 64x32 output tile with its halo is staged in shared memory once, filtered along x into a
// second shared tile, then along y into registers; each thread produces 8 outputs from a
// sliding window so a tap costs ~1/4 shared-memory word.  The threshold kernel evaluates
// eq. 5 with the S_eff guard, tests eq. 6 lazily (only for pixels that passed eq. 5) and
// appends eq. 7 peaks with one atomic per warp.
#include "lpf_internal.cuh"

namespace {

constexpr int TX = 64, TY = 32, CT = 256;

enum { MODE_MF = 0, MODE_C = 1, MODE_S = 2, MODE_DEN = 3 };

struct ConvArgs {
  const float* src;       // MODE_MF: cube ; MODE_C / MODE_S: F planes ; MODE_DEN: unused
  const float* src_sum;   // MODE_MF: the sum plane (plane B)
  const float* Cpl;       // MODE_S: C planes
  const uint8_t* W;       // [N]
  const uint8_t* Y;       // [(B+1)][N] or null
  const float* norm;      // [N] (or [(B+1)][N] if norm_per_plane)
  float* out;             // [(B+1)][N]   (MODE_DEN on the static mask: [N])
  const uint8_t* band_ok; // null: every plane active (static precomputation)
  int norm_per_plane;
  int B, Dy, Dx, n_planes;
  LpfTaps g;
};

__device__ __forceinline__ bool plane_active(const uint8_t* band_ok, int B, int p) {
  if (!band_ok) return true;
  if (!band_ok[B]) return false;
  return p >= B ? true : band_ok[p] != 0;
}

template <int MODE>
__device__ __forceinline__ float load_in(const ConvArgs& a, const float* src_p, const float* C_p,
                                         const uint8_t* Y_p, int y, int x) {
  if (y < 0 || y >= a.Dy || x < 0 || x >= a.Dx) return 0.f;
  const long long q = (long long)y * a.Dx + x;
  bool w = a.W[q] != 0;
  if (MODE != MODE_MF && Y_p) w = w && (Y_p[q] == 0);
  if (!w) return 0.f;
  if (MODE == MODE_DEN) return 1.f;
  const float v = src_p[q];
  if (MODE == MODE_S) { const float d = v - C_p[q]; return d * d; }
  return v;
}

// RT > 0: compile-time radius (sliding-window FMAs on registers); RT == 0: run-time radius.
template <int MODE, int RT>
__global__ void __launch_bounds__(CT)
k_sepconv(const ConvArgs a) {
  extern __shared__ float sm[];
  const int R = RT > 0 ? RT : a.g.R;
  const int p = blockIdx.z;
  if (!plane_active(a.band_ok, a.B, p)) return;
  const long long N = (long long)a.Dy * a.Dx;
  const int TYH = TY + 2 * R;
  const int PIN = (TX + 2 * R) | 1;
  const int PT = TX + 1;
  float* s_in = sm;
  float* s_tmp = sm + TYH * PIN;
  const float* src_p = nullptr;
  if (MODE == MODE_MF) src_p = (p < a.B) ? a.src + (long long)p * N : a.src_sum;
  else if (MODE != MODE_DEN) src_p = a.src + (long long)p * N;
  const float* C_p = (MODE == MODE_S) ? a.Cpl + (long long)p * N : nullptr;
  const uint8_t* Y_p = (a.Y && MODE != MODE_MF) ? a.Y + (long long)p * N : nullptr;
  const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY;

  for (int i = threadIdx.x; i < TYH * (TX + 2 * R); i += CT) {
    const int r = i / (TX + 2 * R), cc = i - r * (TX + 2 * R);
    s_in[r * PIN + cc] = load_in<MODE>(a, src_p, C_p, Y_p, y0 - R + r, x0 - R + cc);
  }
  __syncthreads();

  // row pass: lanes <-> consecutive rows (odd pitch: conflict-free), 8 outputs per item
  for (int it = threadIdx.x; it < TYH * (TX / 8); it += CT) {
    const int r = it % TYH, cg = it / TYH;
    const float* row = s_in + r * PIN + cg * 8;
    float acc[8];
#pragma unroll
    for (int o = 0; o < 8; ++o) acc[o] = 0.f;
    if (RT > 0) {
      float v[8 + 2 * (RT > 0 ? RT : 1)];
#pragma unroll
      for (int i = 0; i < 8 + 2 * RT; ++i) v[i] = row[i];
#pragma unroll
      for (int o = 0; o < 8; ++o)
#pragma unroll
        for (int i = 0; i <= 2 * RT; ++i) acc[o] = fmaf(a.g.g[i], v[o + i], acc[o]);
    } else {
      for (int i = 0; i <= 2 * R; ++i) {
        const float gi = a.g.g[i];
#pragma unroll
        for (int o = 0; o < 8; ++o) acc[o] = fmaf(gi, row[o + i], acc[o]);
      }
    }
#pragma unroll
    for (int o = 0; o < 8; ++o) s_tmp[r * PT + cg * 8 + o] = acc[o];
  }
  __syncthreads();

  // column pass: lanes <-> consecutive columns, 8 output rows per thread
  {
    const int cx = threadIdx.x % TX, rg = threadIdx.x / TX;  // rg in 0..3
    const float* col = s_tmp + (rg * 8) * PT + cx;
    float acc[8];
#pragma unroll
    for (int o = 0; o < 8; ++o) acc[o] = 0.f;
    if (RT > 0) {
      float v[8 + 2 * (RT > 0 ? RT : 1)];
#pragma unroll
      for (int j = 0; j < 8 + 2 * RT; ++j) v[j] = col[j * PT];
#pragma unroll
      for (int o = 0; o < 8; ++o)
#pragma unroll
        for (int j = 0; j <= 2 * RT; ++j) acc[o] = fmaf(a.g.g[j], v[o + j], acc[o]);
    } else {
      for (int j = 0; j <= 2 * R; ++j) {
        const float gj = a.g.g[j];
#pragma unroll
        for (int o = 0; o < 8; ++o) acc[o] = fmaf(gj, col[(o + j) * PT], acc[o]);
      }
    }
    const int x = x0 + cx;
    if (x < a.Dx) {
#pragma unroll
      for (int o = 0; o < 8; ++o) {
        const int y = y0 + rg * 8 + o;
        if (y >= a.Dy) break;
        const long long q = (long long)y * a.Dx + x;
        float r;
        if (MODE == MODE_DEN) {
          r = (a.W[q] && acc[o] > 0.f) ? 1.0f / acc[o] : 0.f;
        } else {
          const float nm = a.norm_per_plane ? a.norm[(long long)p * N + q] : a.norm[q];
          r = acc[o] * nm;
        }
        a.out[(MODE == MODE_DEN && !a.band_ok) ? q : (long long)p * N + q] = r;
      }
    }
  }
}

template <int MODE>
int launch_sepconv(lpf_ctx* c, const ConvArgs& a, cudaStream_t st) {
  const int R = a.g.R;
  const dim3 grid((a.Dx + TX - 1) / TX, (a.Dy + TY - 1) / TY, a.n_planes);
  const size_t smem = (size_t)((TY + 2 * R) * (((TX + 2 * R) | 1) + (TX + 1))) * sizeof(float);
  const int kid = MODE == MODE_MF ? KID_CONV_MF : MODE == MODE_C ? KID_CONV_C : MODE == MODE_S ? KID_CONV_S : KID_CONV_DEN;
  switch (R) {
    case 3: LPF_KLAUNCH(c, kid, st, k_sepconv<MODE, 3><<<grid, CT, smem, st>>>(a)); break;
    case 12: LPF_KLAUNCH(c, kid, st, k_sepconv<MODE, 12><<<grid, CT, smem, st>>>(a)); break;
    case 16: LPF_KLAUNCH(c, kid, st, k_sepconv<MODE, 16><<<grid, CT, smem, st>>>(a)); break;
    default: LPF_KLAUNCH(c, kid, st, k_sepconv<MODE, 0><<<grid, CT, smem, st>>>(a)); break;
  }
  return LPF_OK;
}

struct ThrArgs {
  const float* F; const float* C; const float* S;
  const uint8_t* W; uint8_t* Y; const uint8_t* band_ok;
  int B, Dy, Dx, k_max, iter, max_det;
  float kappa2, eps_rel;
  lpf_det* dets; int32_t* ndets; int32_t* counters;
};

// eq. 5 (+ guard R8), eq. 6 lazily, eq. 7, warp-aggregated append.
__global__ void __launch_bounds__(256)
k_threshold_peaks(const ThrArgs a) {
  const int p = blockIdx.z;
  if (!plane_active(a.band_ok, a.B, p)) return;
  const long long N = (long long)a.Dy * a.Dx;
  const long long pix = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const float* F = a.F + (long long)p * N;
  bool peak = false;
  float f = 0.f, cc = 0.f, se = 0.f, d = 0.f;
  if (pix < N && a.W[pix] && !(a.Y && a.Y[(long long)p * N + pix])) {
    f = F[pix]; cc = a.C[(long long)p * N + pix];
    const float s = a.S[(long long)p * N + pix];
    d = f - cc;
    const float gd = a.eps_rel * fabsf(cc);
    se = fmaxf(s, gd * gd);
    if (d > 0.f && d * d > a.kappa2 * se) {
      if (a.Y) a.Y[(long long)p * N + pix] = (uint8_t)a.iter;
      peak = true;
      const int y = (int)(pix / a.Dx), x = (int)(pix - (long long)y * a.Dx);
      for (int j = -a.k_max; j <= a.k_max && peak; ++j) {
        const int yy = y + j;
        if (yy < 0 || yy >= a.Dy) continue;
        for (int i = -a.k_max; i <= a.k_max; ++i) {
          const int xx = x + i;
          if (xx < 0 || xx >= a.Dx) continue;
          const long long q = (long long)yy * a.Dx + xx;
          if (a.W[q] && F[q] > f) { peak = false; break; }
        }
      }
    }
  }
  const unsigned m = __ballot_sync(0xffffffffu, peak);
  if (m) {
    const int lane = threadIdx.x & 31;
    int base = 0;
    if (lane == (__ffs(m) - 1)) base = atomicAdd(a.ndets, __popc(m));
    base = __shfl_sync(0xffffffffu, base, __ffs(m) - 1);
    if (peak) {
      const int idx = base + __popc(m & ((1u << lane) - 1u));
      if (idx < a.max_det) {
        lpf_det r;
        r.pix = (int32_t)pix; r.plane = (int16_t)p; r.iter = (int16_t)a.iter;
        r.f = f; r.c = cc; r.s = se; r.snr = d / sqrtf(se);
        a.dets[idx] = r;
      } else {
        atomicAdd(&a.counters[0], 1);
      }
    }
  }
}

}  // namespace

// norm = W / (g (*) W) for the static mask (R7).  d_tmp unused (kept for symmetry).
int lpf_launch_static_norm(lpf_ctx* c, const LpfTaps& g, float* d_norm, float* /*d_tmp*/, cudaStream_t st) {
  ConvArgs a{};
  a.W = c->W; a.Y = nullptr; a.out = d_norm; a.band_ok = nullptr;
  a.B = c->p.B; a.Dy = c->p.Dy; a.Dx = c->p.Dx; a.n_planes = 1; a.g = g;
  return launch_sepconv<MODE_DEN>(c, a, st);
}

int lpf_launch_detect_general(lpf_ctx* c, LpfLane& L, const float* d_cube, const uint8_t* d_band_ok,
                              lpf_det* d_dets, int32_t* d_ndets, bool sum_done, cudaStream_t st) {
  const lpf_params& p = c->p;
  int rc;
  if (!sum_done) {
    LPF_CUDA(cudaMemsetAsync(d_ndets, 0, sizeof(int32_t), st));
    if (p.detect_sum_plane) { rc = lpf_launch_sum_plane(c, L, d_cube, d_band_ok, true, st); if (rc) return rc; }
  }
  if (p.n_iter > 1) LPF_CUDA(cudaMemsetAsync(L.Y, 0, (size_t)c->n_planes * c->N, st));

  ConvArgs a{};
  a.W = c->W; a.band_ok = d_band_ok; a.B = p.B; a.Dy = p.Dy; a.Dx = p.Dx; a.n_planes = c->n_planes;
  // S4: matched filter
  a.src = d_cube; a.src_sum = L.sum_plane; a.Y = nullptr; a.norm = c->norm_mf; a.norm_per_plane = 0;
  a.out = L.F; a.g = c->g_mf;
  rc = launch_sepconv<MODE_MF>(c, a, st); if (rc) return rc;

  for (int it = 1; it <= p.n_iter; ++it) {
    a.g = c->g_bg; a.src = L.F; a.src_sum = nullptr;
    a.Y = (it > 1) ? L.Y : nullptr;
    if (it > 1) {  // denominators of W' = W and not Y, per plane
      a.out = L.normp; a.norm = nullptr; a.norm_per_plane = 0;
      rc = launch_sepconv<MODE_DEN>(c, a, st); if (rc) return rc;
      a.norm = L.normp; a.norm_per_plane = 1;
    } else {
      a.norm = c->norm_bg; a.norm_per_plane = 0;
    }
    a.out = L.C;                                   // S5: C = G (*)_W' F          (eq. 3)
    rc = launch_sepconv<MODE_C>(c, a, st); if (rc) return rc;
    a.Cpl = L.C; a.out = L.S;                      //     S = G (*)_W' (F-C)^2    (eq. 4)
    rc = launch_sepconv<MODE_S>(c, a, st); if (rc) return rc;

    ThrArgs t{};                                   // S6-S8
    t.F = L.F; t.C = L.C; t.S = L.S; t.W = c->W; t.Y = (p.n_iter > 1) ? L.Y : nullptr; t.band_ok = d_band_ok;
    t.B = p.B; t.Dy = p.Dy; t.Dx = p.Dx; t.k_max = p.k_max; t.iter = it; t.max_det = p.max_det;
    t.kappa2 = p.kappa * p.kappa; t.eps_rel = p.eps_rel;
    t.dets = d_dets; t.ndets = d_ndets; t.counters = c->counters;
    const dim3 grid((unsigned)((c->N + 255) / 256), 1, c->n_planes);
    LPF_KLAUNCH(c, KID_THRESHOLD, st, k_threshold_peaks<<<grid, 256, 0, st>>>(t));
  }
  return LPF_OK;
}
