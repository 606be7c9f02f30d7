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

// ---- the wide form: radius 3 (matched filter), 12 or 16 on images whose rows are whole float4 groups ---------------
// A 128 x 64 output tile (halo amplification 1.9 instead of 3 at radius 16).  Staging: a thread loads the same float4
// group of two tile rows half a tile apart (mask word, values, for the spread also C: all loads of a round issued
// before the first is used) and stores the two rows interleaved, so that one 128-bit shared load in the row pass
// gives two ready f32x2 pairs (lanes <-> consecutive row pairs, pitch chosen for conflict-free 128-bit loads).  The
// column pass pairs two neighbouring columns.  Both passes are packed FFMA2 with the taps applied in the same order
// as in k_sepconv, so the two forms give the same bits.  RL: the halo staged (a multiple of 4 >= R: groups stay
// aligned).
constexpr int WTX = 128, WTY = 64, WPIN = 162, WPT = 132;

template <int MODE>
__device__ __forceinline__ float4 wide_value(float4 v, float4 cv, unsigned w) {
  if (MODE == MODE_DEN) v = make_float4(1.f, 1.f, 1.f, 1.f);
  if (MODE == MODE_S) {
    const float d0 = v.x - cv.x, d1 = v.y - cv.y, d2 = v.z - cv.z, d3 = v.w - cv.w;
    v = make_float4(d0 * d0, d1 * d1, d2 * d2, d3 * d3);
  }
  if (!(w & 0x000000ffu)) v.x = 0.f;      // selects, not products: an invalid pixel may hold anything
  if (!(w & 0x0000ff00u)) v.y = 0.f;
  if (!(w & 0x00ff0000u)) v.z = 0.f;
  if (!(w & 0xff000000u)) v.w = 0.f;
  return v;
}

__device__ __forceinline__ unsigned wide_mask(unsigned w, unsigned yy) {     // W and not Y, per byte
  if (yy & 0x000000ffu) w &= ~0x000000ffu;
  if (yy & 0x0000ff00u) w &= ~0x0000ff00u;
  if (yy & 0x00ff0000u) w &= ~0x00ff0000u;
  if (yy & 0xff000000u) w &= ~0xff000000u;
  return w;
}

template <int MODE, int R, int RL>
__global__ void __launch_bounds__(CT, 2)
k_sepconv_wide(const ConvArgs a) {
  extern __shared__ float4 sm4[];
  constexpr int TYH = WTY + 2 * RL, NG = (WTX + 2 * RL) / 4, HALF = TYH / 2, OFF = RL - R;
  static_assert(RL % 4 == 0 && RL >= R && RL <= 16 && 4 * NG <= WPIN, "wide form: staged halo");
  float* s_in = reinterpret_cast<float*>(sm4);      // [HALF][WPIN] pairs: (row r, row r + HALF)
  float* s_tmp = s_in + TYH * WPIN;                 // [TYH][WPT]
  const int p = blockIdx.z;
  if (!plane_active(a.band_ok, a.B, p)) return;
  const long long N = (long long)a.Dy * a.Dx;
  const float* src_p = nullptr;
  if (MODE == MODE_MF) src_p = (p < a.B) ? a.src + (long long)p * N : a.src_sum;
  else if (MODE != MODE_DEN) src_p = a.src + (long long)p * N;
  const float* C_p = (MODE == MODE_S) ? a.Cpl + (long long)p * N : nullptr;
  const uint8_t* Y_p = (a.Y && MODE != MODE_MF) ? a.Y + (long long)p * N : nullptr;
  const int x0 = blockIdx.x * WTX, y0 = blockIdx.y * WTY;

  // staging: items (row pair, group), WU items per round (the spread also holds C: half as many)
#ifndef LPF_WU_BIG
#define LPF_WU_BIG 8
#endif
  constexpr int WU = (MODE == MODE_S) ? 4 : LPF_WU_BIG;
  for (int i0 = threadIdx.x; i0 < HALF * NG; i0 += WU * CT) {
    unsigned w[WU][2];
    float4 v[WU][2], cv[WU][2];
    long long q[WU][2];
    bool in[WU][2];
#pragma unroll
    for (int u = 0; u < WU; ++u) {
      const int i = i0 + u * CT;
      const int r = i / NG, g = i - r * NG;
      const int x = x0 - RL + 4 * g;
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const int y = y0 - RL + r + h * HALF;
        in[u][h] = i < HALF * NG && y >= 0 && y < a.Dy && x >= 0 && x < a.Dx;   // Dx % 4 == 0: a group is inside or outside as a whole
        q[u][h] = in[u][h] ? (long long)y * a.Dx + x : 0;
        w[u][h] = in[u][h] ? __ldg(reinterpret_cast<const unsigned*>(a.W + q[u][h])) : 0u;
      }
    }
    if (Y_p) {
#pragma unroll
      for (int u = 0; u < WU; ++u)
#pragma unroll
        for (int h = 0; h < 2; ++h)
          if (in[u][h]) w[u][h] = wide_mask(w[u][h], *reinterpret_cast<const unsigned*>(Y_p + q[u][h]));
    }
#pragma unroll
    for (int u = 0; u < WU; ++u)
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        v[u][h] = make_float4(0.f, 0.f, 0.f, 0.f); cv[u][h] = v[u][h];
        if (MODE != MODE_DEN && in[u][h]) v[u][h] = *reinterpret_cast<const float4*>(src_p + q[u][h]);
        if (MODE == MODE_S && in[u][h]) cv[u][h] = *reinterpret_cast<const float4*>(C_p + q[u][h]);
      }
#pragma unroll
    for (int u = 0; u < WU; ++u) {
      const int i = i0 + u * CT;
      if (i < HALF * NG) {
        const int r = i / NG, g = i - r * NG;
        const float4 va = wide_value<MODE>(v[u][0], cv[u][0], w[u][0]), vb = wide_value<MODE>(v[u][1], cv[u][1], w[u][1]);
        float4* dst = reinterpret_cast<float4*>(s_in + 2 * (r * WPIN + 4 * g));
        dst[0] = make_float4(va.x, vb.x, va.y, vb.y);
        dst[1] = make_float4(va.z, vb.z, va.w, vb.w);
      }
    }
  }
  __syncthreads();

  // row pass: an item = rows (r, r + HALF) x 8 output columns
  for (int it = threadIdx.x; it < HALF * (WTX / 8); it += CT) {
    const int r = it % HALF, cg = it / HALF;
    const float* rp = s_in + 2 * (r * WPIN + cg * 8 + OFF);
    float2 v[8 + 2 * R];
    if (OFF % 2 == 0) {
#pragma unroll
      for (int i = 0; i < (8 + 2 * R) / 2; ++i) {
        const float4 x2 = reinterpret_cast<const float4*>(rp)[i];
        v[2 * i] = make_float2(x2.x, x2.y); v[2 * i + 1] = make_float2(x2.z, x2.w);
      }
    } else {
#pragma unroll
      for (int i = 0; i < 8 + 2 * R; ++i) v[i] = reinterpret_cast<const float2*>(rp)[i];
    }
    float2 acc[8];
#pragma unroll
    for (int o = 0; o < 8; ++o) {
      acc[o] = make_float2(0.f, 0.f);
#pragma unroll
      for (int i = 0; i <= 2 * R; ++i) acc[o] = __ffma2_rn(make_float2(a.g.g[i], a.g.g[i]), v[o + i], acc[o]);
    }
    float4* oa = reinterpret_cast<float4*>(s_tmp + r * WPT + cg * 8);
    float4* ob = reinterpret_cast<float4*>(s_tmp + (r + HALF) * WPT + cg * 8);
    oa[0] = make_float4(acc[0].x, acc[1].x, acc[2].x, acc[3].x); oa[1] = make_float4(acc[4].x, acc[5].x, acc[6].x, acc[7].x);
    ob[0] = make_float4(acc[0].y, acc[1].y, acc[2].y, acc[3].y); ob[1] = make_float4(acc[4].y, acc[5].y, acc[6].y, acc[7].y);
  }
  __syncthreads();

  // column pass: a thread = columns (2 cp, 2 cp + 1) x 16 output rows, in two blocks of 8
  {
    const int cp = threadIdx.x % (WTX / 2), rg = threadIdx.x / (WTX / 2);   // rg in 0..3
    const int x = x0 + 2 * cp;
#pragma unroll 1
    for (int blk = 0; blk < 2; ++blk) {
      const int ry = rg * 16 + blk * 8;
      const float* col = s_tmp + (ry + OFF) * WPT + 2 * cp;
      float2 v[8 + 2 * R];
#pragma unroll
      for (int j = 0; j < 8 + 2 * R; ++j) v[j] = *reinterpret_cast<const float2*>(col + j * WPT);
      float2 acc[8];
#pragma unroll
      for (int o = 0; o < 8; ++o) {
        acc[o] = make_float2(0.f, 0.f);
#pragma unroll
        for (int j = 0; j <= 2 * R; ++j) acc[o] = __ffma2_rn(make_float2(a.g.g[j], a.g.g[j]), v[o + j], acc[o]);
      }
      if (x < a.Dx) {
#pragma unroll
        for (int o = 0; o < 8; ++o) {
          const int y = y0 + ry + o;
          if (y >= a.Dy) break;
          const long long q = (long long)y * a.Dx + x;
          float2 r;
          if (MODE == MODE_DEN) {
            const uint8_t w0 = a.W[q], w1 = a.W[q + 1];
            r.x = (w0 && acc[o].x > 0.f) ? 1.0f / acc[o].x : 0.f;
            r.y = (w1 && acc[o].y > 0.f) ? 1.0f / acc[o].y : 0.f;
          } else {
            const float2 nm = *reinterpret_cast<const float2*>(a.norm + (a.norm_per_plane ? (long long)p * N + q : q));
            r.x = acc[o].x * nm.x; r.y = acc[o].y * nm.y;
          }
          *reinterpret_cast<float2*>(a.out + ((MODE == MODE_DEN && !a.band_ok) ? q : (long long)p * N + q)) = r;
        }
      }
    }
  }
}

template <int R> struct WideHalo { static constexpr int RL = (R + 3) / 4 * 4; };

template <int MODE, int R>
cudaError_t sepconv_wide_attr() {
  constexpr int RL = WideHalo<R>::RL;
  constexpr size_t smem = (size_t)(WTY + 2 * RL) * (WPIN + WPT) * sizeof(float);
  return cudaFuncSetAttribute(k_sepconv_wide<MODE, R, RL>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
}

template <int MODE, int R>
int launch_sepconv_wide(lpf_ctx* c, int kid, const ConvArgs& a, cudaStream_t st) {
  constexpr int RL = WideHalo<R>::RL;
  constexpr size_t smem = (size_t)(WTY + 2 * RL) * (WPIN + WPT) * sizeof(float);
  const dim3 grid((a.Dx + WTX - 1) / WTX, (a.Dy + WTY - 1) / WTY, a.n_planes);
  LPF_KLAUNCH(c, kid, st, k_sepconv_wide<MODE, R, RL><<<grid, CT, smem, st>>>(a));
  return LPF_OK;
}

template <int MODE>
int launch_sepconv(lpf_ctx* c, const ConvArgs& a, cudaStream_t st) {
  const int R = a.g.R;
  const int kid = MODE == MODE_MF ? KID_CONV_MF : MODE == MODE_C ? KID_CONV_C : MODE == MODE_S ? KID_CONV_S : KID_CONV_DEN;
  // the wide form loads 128 bits at a time: rows of whole groups, and a caller's cube on a 16-byte boundary
  const bool al16 = (reinterpret_cast<uintptr_t>(a.src) & 15u) == 0 && (reinterpret_cast<uintptr_t>(a.src_sum) & 15u) == 0;
  if (a.Dx % 4 == 0 && al16) {
    if (R == 3) return launch_sepconv_wide<MODE, 3>(c, kid, a, st);
    if (R == 12) return launch_sepconv_wide<MODE, 12>(c, kid, a, st);
    if (R == 16) return launch_sepconv_wide<MODE, 16>(c, kid, a, st);
  }
  const dim3 grid((a.Dx + TX - 1) / TX, (a.Dy + TY - 1) / TY, a.n_planes);
  const size_t smem = (size_t)((TY + 2 * R) * (((TX + 2 * R) | 1) + (TX + 1))) * sizeof(float);
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

// The same for four pixels per thread (N % 4 == 0, Dx % 4 == 0): 128-bit loads of F, C, S, word loads of W and Y.
// Eq. 6 is tested by the warp together: for every pixel of the warp that passed eq. 5, lane l looks at neighbour l of
// the (2 k_max + 1)^2 window (in rounds of 32), so a hit costs the warp a dozen instructions instead of a serial loop.
__global__ void __launch_bounds__(256)
k_threshold_peaks4(const ThrArgs a) {
  const int p = blockIdx.z;
  if (!plane_active(a.band_ok, a.B, p)) return;
  const long long N = (long long)a.Dy * a.Dx;
  const long long pix0 = 4 * ((long long)blockIdx.x * blockDim.x + threadIdx.x);
  const float* F = a.F + (long long)p * N;
  const int lane = threadIdx.x & 31;
  unsigned hits = 0u, peaks = 0u;
  // eq. 5 for the thread's four pixels without a branch: nothing but the three loaded vectors stays live; the few
  // threads with a hit work their record values out again below
  float4 f4 = make_float4(0.f, 0.f, 0.f, 0.f), c4 = f4, s4 = f4;
  if (pix0 < N) {
    unsigned w = *reinterpret_cast<const unsigned*>(a.W + pix0);
    unsigned yy = 0u;
    if (a.Y) { yy = *reinterpret_cast<const unsigned*>(a.Y + (long long)p * N + pix0); w = wide_mask(w, yy); }
    if (w) {
      f4 = *reinterpret_cast<const float4*>(F + pix0);
      c4 = *reinterpret_cast<const float4*>(a.C + (long long)p * N + pix0);
      s4 = *reinterpret_cast<const float4*>(a.S + (long long)p * N + pix0);
      const float fv[4] = {f4.x, f4.y, f4.z, f4.w}, cv[4] = {c4.x, c4.y, c4.z, c4.w}, sv[4] = {s4.x, s4.y, s4.z, s4.w};
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const float dk = fv[k] - cv[k];
        const float gd = a.eps_rel * fabsf(cv[k]);
        const float sek = fmaxf(sv[k], gd * gd);
        const bool h = ((w >> (8 * k)) & 0xffu) != 0u && dk > 0.f && dk * dk > a.kappa2 * sek;
        hits |= h ? (1u << k) : 0u;
      }
      if (a.Y && hits) {
        unsigned ynew = yy;
#pragma unroll
        for (int k = 0; k < 4; ++k) if ((hits >> k) & 1u) ynew |= (unsigned)(a.iter & 0xff) << (8 * k);
        *reinterpret_cast<unsigned*>(a.Y + (long long)p * N + pix0) = ynew;
      }
    }
  }
  if (!__any_sync(0xffffffffu, hits != 0u)) return;
  float f[4], cc[4], se[4], d[4];
  {
    const float fv[4] = {f4.x, f4.y, f4.z, f4.w}, cv[4] = {c4.x, c4.y, c4.z, c4.w}, sv[4] = {s4.x, s4.y, s4.z, s4.w};
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      f[k] = fv[k]; cc[k] = cv[k];
      d[k] = f[k] - cc[k];
      const float gd = a.eps_rel * fabsf(cc[k]);
      se[k] = fmaxf(sv[k], gd * gd);
    }
  }
  const int side = 2 * a.k_max + 1, nwin = side * side;
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    unsigned m = __ballot_sync(0xffffffffu, (hits >> k) & 1u);
    while (m) {
      const int src = __ffs(m) - 1;
      m &= m - 1;
      const long long pix = __shfl_sync(0xffffffffu, pix0, src) + k;
      const float fc = __shfl_sync(0xffffffffu, f[k], src);
      const int y = (int)(pix / a.Dx), x = (int)(pix - (long long)y * a.Dx);
      bool beaten = false;
      for (int n0 = 0; n0 < nwin; n0 += 32) {
        const int n = n0 + lane;
        if (n < nwin) {
          const int yq = y + n / side - a.k_max, xx = x + n % side - a.k_max;
          if (yq >= 0 && yq < a.Dy && xx >= 0 && xx < a.Dx) {
            const long long q = (long long)yq * a.Dx + xx;
            beaten = beaten || (a.W[q] && F[q] > fc);
          }
        }
      }
      if (!__any_sync(0xffffffffu, beaten) && lane == src) peaks |= 1u << k;
    }
  }
  if (!__any_sync(0xffffffffu, peaks != 0u)) return;
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    const bool peak = (peaks >> k) & 1u;
    const unsigned m = __ballot_sync(0xffffffffu, peak);
    if (!m) continue;
    int base = 0;
    if (lane == (__ffs(m) - 1)) base = atomicAdd(a.ndets, __popc(m));
    base = __shfl_sync(0xffffffffu, base, __ffs(m) - 1);
    if (peak) {
      const int idx = base + __popc(m & ((1u << lane) - 1u));
      if (idx < a.max_det) {
        lpf_det r;
        r.pix = (int32_t)(pix0 + k); r.plane = (int16_t)p; r.iter = (int16_t)a.iter;
        r.f = f[k]; r.c = cc[k]; r.s = se[k]; r.snr = d[k] / sqrtf(se[k]);
        a.dets[idx] = r;
      } else {
        atomicAdd(&a.counters[0], 1);
      }
    }
  }
}

}  // namespace

// kernel attributes of the wide form, once per process, outside any stream capture (lpf_create)
int lpf_general_prepare(void) {
#define LPF_WIDE_ATTR(M) LPF_CUDA((sepconv_wide_attr<M, 3>())); LPF_CUDA((sepconv_wide_attr<M, 12>())); LPF_CUDA((sepconv_wide_attr<M, 16>()));
  LPF_WIDE_ATTR(MODE_MF) LPF_WIDE_ATTR(MODE_C) LPF_WIDE_ATTR(MODE_S) LPF_WIDE_ATTR(MODE_DEN)
#undef LPF_WIDE_ATTR
  return LPF_OK;
}

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
    if (p.Dx % 4 == 0) {
      const dim3 grid((unsigned)((c->N / 4 + 255) / 256), 1, c->n_planes);
      LPF_KLAUNCH(c, KID_THRESHOLD, st, k_threshold_peaks4<<<grid, 256, 0, st>>>(t));
    } else {
      const dim3 grid((unsigned)((c->N + 255) / 256), 1, c->n_planes);
      LPF_KLAUNCH(c, KID_THRESHOLD, st, k_threshold_peaks<<<grid, 256, 0, st>>>(t));
    }
  }
  return LPF_OK;
}
