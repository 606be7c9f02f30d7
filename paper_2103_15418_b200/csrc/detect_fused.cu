// S4-S8 fused fast path: matched filter -> local centre -> local spread -> sigma clip -> local
// maxima -> compaction in ONE pass over each plane, for the headline parameter set
// (box background K = 12, Gaussian matched filter k_mf = 3, n_iter = 1).
// (eqs. 2-7; O3-O6 and "Fused detection kernel".)
//
// Design (sm_100a): a CTA owns a column strip (as wide as shared memory allows: the two 26-row
// ring buffers of a whole 922-column all-sky strip fit the 227 KB of one SM) and sweeps down a
// segment of rows.  Each thread owns 4 adjacent columns and RB rows per iteration:
//   A  128-bit global loads of X (masked by W)                                   [HBM/L2]
//   B  horizontal 7-tap matched filter (neighbour groups through shared memory)
//   C  vertical 7-tap matched filter on a register window, x norm_mf  -> F
//   D  vertical 25-row running sum of F (ring buffer of F rows in shared memory)
//   E  horizontal 25-box of the running sums by blocked partial sums, x 1/count -> C   (eq. 3)
//   F  d = F - C (F re-read from the ring at lag 12)
//   G  vertical 25-row running sum of d^2 (ring buffer of d rows)
//   H  horizontal 25-box, x 1/count                                             -> S   (eq. 4)
//   I  eq. 5 on d at lag 12; only pixels that pass take the slow path: S_eff guard, eq. 6
//      local-maximum test on the F ring, eq. 7 record with a warp-aggregated atomic.
// F, C, d and S never leave the SM.  The dependent double stencil costs 27 warm-up rows per
// segment and no redundant columns when the strip spans the valid width of the image.
#include <algorithm>
#include <cstdio>
#include <cstdlib>

#include "lpf_internal.cuh"

namespace {

constexpr int RBF = 2;         // rows per iteration
constexpr int KBG = 12;        // box half width
constexpr int WINB = 2 * KBG + 1;
constexpr int DF = WINB + 1 + RBF;  // F ring depth: lag 25 (running sum) .. lag 26 (local max) + rows in flight
constexpr int DD = WINB + 1;        // d ring depth

struct FusedItem { int xs, ux0, ux1, ya, yb; };

struct FusedArgs {
  const float* cube; const float* sum_plane; const uint8_t* band_ok; const uint8_t* W;
  const float* norm_mf; const float* inv_cnt; const FusedItem* items;
  int B, Dy, Dx, CW, k_max, max_det;
  float g0, g1, g2, g3, kappa2, eps_rel;
  lpf_det* dets; int32_t* ndets; int32_t* counters;
};

__device__ __forceinline__ float4 ld4(const float* p) { return *reinterpret_cast<const float4*>(p); }
__device__ __forceinline__ void st4(float* p, const float4 v) { *reinterpret_cast<float4*>(p) = v; }
__device__ __forceinline__ float4 ldg4(const float* p) { return __ldg(reinterpret_cast<const float4*>(p)); }

__device__ __forceinline__ int wrap_add(int a, int b, int m) { const int s = a + b; return s >= m ? s - m : s; }

// horizontal 25-box of one row of per-column values held 4 per thread (own = v, group sum = t)
__device__ __forceinline__ void hbox25(const float* EVrow, const float* ETrow, int tid, float t, float out[4]) {
  const float tm2 = ETrow[tid], tm1 = ETrow[tid + 1], tp1 = ETrow[tid + 3], tp2 = ETrow[tid + 4];
  const float4 L = ld4(EVrow + 4 * tid);        // group q-3
  const float4 R = ld4(EVrow + 4 * tid + 24);   // group q+3
  const float g5 = ((tm2 + tm1) + t) + (tp1 + tp2);
  const float sL = (L.x + L.y) + (L.z + L.w);
  out[0] = (g5 + sL) + R.x;
  out[1] = out[0] + (R.y - L.x);
  out[2] = out[1] + (R.z - L.y);
  out[3] = out[2] + (R.w - L.z);
}

__global__ void __launch_bounds__(256, 1)
k_fused_box(const FusedArgs a) {
  extern __shared__ float4 sm4[];
  float* sm = reinterpret_cast<float*>(sm4);
  const int p = blockIdx.y;
  if (!a.band_ok[a.B]) return;
  if (p < a.B && !a.band_ok[p]) return;
  const FusedItem it = a.items[blockIdx.x];
  const int CW = a.CW, tid = threadIdx.x;
  const int PEX = CW + 8, PEV = CW + 24, PET = CW / 4 + 4;
  float* ringF = sm;
  float* ringD = ringF + DF * CW;
  float* EX = ringD + DD * CW;
  float* EV = EX + RBF * PEX;
  float* EV2 = EV + RBF * PEV;
  float* ET = EV2 + RBF * PEV;
  float* ET2 = ET + RBF * PET;
  const int total = (DF + DD) * CW + RBF * (PEX + 2 * PEV + 2 * PET);
  for (int i = tid; i < total; i += blockDim.x) sm[i] = 0.f;
  __syncthreads();

  const long long N = (long long)a.Dy * a.Dx;
  const float* X = (p < a.B) ? a.cube + (long long)p * N : a.sum_plane;
  const int x = it.xs + 4 * tid;
  const bool col_in = x < a.Dx;
  const float g0 = a.g0, g1 = a.g1, g2 = a.g2, g3 = a.g3;

  float hw[6 + RBF][4];
#pragma unroll
  for (int i = 0; i < 6 + RBF; ++i)
#pragma unroll
    for (int k = 0; k < 4; ++k) hw[i][k] = 0.f;
  float V1[4] = {0.f, 0.f, 0.f, 0.f}, V2[4] = {0.f, 0.f, 0.f, 0.f};

  const int y_start = it.ya - (2 * KBG + 3);
  const int nb = (it.yb - it.ya + 2 * (2 * KBG + 3) + RBF - 1) / RBF;
  int wF = 0, wD = 0;  // ring slots of the next F row / next d row

  for (int b = 0; b < nb; ++b) {
    const int yb0 = y_start + b * RBF;
    // ---- A: load, mask; B: horizontal matched filter -----------------------------------
    float xm[RBF][4];
#pragma unroll
    for (int j = 0; j < RBF; ++j) {
      const int y = yb0 + j;
      float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
      if (col_in && y >= 0 && y < a.Dy) {
        const long long q = (long long)y * a.Dx + x;
        v = ldg4(X + q);
        const unsigned wm = __ldg(reinterpret_cast<const unsigned*>(a.W + q));
        if (wm != 0x01010101u) {
          if (!(wm & 0x000000ffu)) v.x = 0.f;
          if (!(wm & 0x0000ff00u)) v.y = 0.f;
          if (!(wm & 0x00ff0000u)) v.z = 0.f;
          if (!(wm & 0xff000000u)) v.w = 0.f;
        }
      }
      xm[j][0] = v.x; xm[j][1] = v.y; xm[j][2] = v.z; xm[j][3] = v.w;
      st4(EX + j * PEX + 4 + 4 * tid, v);
    }
    __syncthreads();  // (1)
#pragma unroll
    for (int j = 0; j < RBF; ++j) {
      const float4 L = ld4(EX + j * PEX + 4 * tid);
      const float4 R = ld4(EX + j * PEX + 8 + 4 * tid);
      const float v[10] = {L.y, L.z, L.w, xm[j][0], xm[j][1], xm[j][2], xm[j][3], R.x, R.y, R.z};
#pragma unroll
      for (int k = 0; k < 4; ++k)
        hw[6 + j][k] = fmaf(g0, v[k + 3], fmaf(g1, v[k + 2] + v[k + 4], fmaf(g2, v[k + 1] + v[k + 5], g3 * (v[k] + v[k + 6]))));
    }
    // ---- C: vertical matched filter -> F rows fr = y - 3 ----------------------------------
    float f[RBF][4];
#pragma unroll
    for (int j = 0; j < RBF; ++j) {
      const int fr = yb0 + j - 3;
      float4 nm = make_float4(0.f, 0.f, 0.f, 0.f);
      if (col_in && fr >= 0 && fr < a.Dy) nm = ldg4(a.norm_mf + (long long)fr * a.Dx + x);
      const float nmv[4] = {nm.x, nm.y, nm.z, nm.w};
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const float acc = fmaf(g0, hw[j + 3][k], fmaf(g1, hw[j + 2][k] + hw[j + 4][k],
                          fmaf(g2, hw[j + 1][k] + hw[j + 5][k], g3 * (hw[j][k] + hw[j + 6][k]))));
        f[j][k] = acc * nmv[k];
      }
    }
#pragma unroll
    for (int i = 0; i < 6; ++i)
#pragma unroll
      for (int k = 0; k < 4; ++k) hw[i][k] = hw[i + RBF][k];
    // ---- D: vertical running sum of F (window fr-24..fr, centre rho = fr-12) ---------------
    float t1[RBF];
#pragma unroll
    for (int j = 0; j < RBF; ++j) {
      const int ws = wrap_add(wF, j, DF);
      const int os = wrap_add(ws, DF - WINB, DF);
      const float4 fo = ld4(ringF + os * CW + 4 * tid);
      V1[0] += f[j][0] - fo.x; V1[1] += f[j][1] - fo.y; V1[2] += f[j][2] - fo.z; V1[3] += f[j][3] - fo.w;
      st4(ringF + ws * CW + 4 * tid, make_float4(f[j][0], f[j][1], f[j][2], f[j][3]));
      st4(EV + j * PEV + 12 + 4 * tid, make_float4(V1[0], V1[1], V1[2], V1[3]));
      t1[j] = (V1[0] + V1[1]) + (V1[2] + V1[3]);
      ET[j * PET + 2 + tid] = t1[j];
    }
    __syncthreads();  // (2)
    // ---- E: C = box / count ; F: d = F - C ; G: running sum of d^2 --------------------------
    float t2[RBF];
#pragma unroll
    for (int j = 0; j < RBF; ++j) {
      const int rho = yb0 + j - 3 - KBG;
      float bx[4];
      hbox25(EV + j * PEV, ET + j * PET, tid, t1[j], bx);
      float4 ic = make_float4(0.f, 0.f, 0.f, 0.f);
      if (col_in && rho >= 0 && rho < a.Dy) ic = ldg4(a.inv_cnt + (long long)rho * a.Dx + x);
      const int ws = wrap_add(wF, j, DF);
      const int rs = wrap_add(ws, DF - KBG, DF);
      const float4 fr4 = ld4(ringF + rs * CW + 4 * tid);
      const float d0 = fr4.x - bx[0] * ic.x, d1 = fr4.y - bx[1] * ic.y, d2 = fr4.z - bx[2] * ic.z, d3 = fr4.w - bx[3] * ic.w;
      const int wd = wrap_add(wD, j, DD);
      const int od = wrap_add(wd, DD - WINB, DD);
      const float4 dold = ld4(ringD + od * CW + 4 * tid);
      V2[0] = fmaf(-dold.x, dold.x, fmaf(d0, d0, V2[0]));
      V2[1] = fmaf(-dold.y, dold.y, fmaf(d1, d1, V2[1]));
      V2[2] = fmaf(-dold.z, dold.z, fmaf(d2, d2, V2[2]));
      V2[3] = fmaf(-dold.w, dold.w, fmaf(d3, d3, V2[3]));
      st4(ringD + wd * CW + 4 * tid, make_float4(d0, d1, d2, d3));
      st4(EV2 + j * PEV + 12 + 4 * tid, make_float4(V2[0], V2[1], V2[2], V2[3]));
      t2[j] = (V2[0] + V2[1]) + (V2[2] + V2[3]);
      ET2[j * PET + 2 + tid] = t2[j];
    }
    __syncthreads();  // (3)
    // ---- H: S = box / count ; I: eq. 5 at sigma = rho - 12 -----------------------------------
#pragma unroll
    for (int j = 0; j < RBF; ++j) {
      const int sg = yb0 + j - 3 - 2 * KBG;
      float bx[4];
      hbox25(EV2 + j * PEV, ET2 + j * PET, tid, t2[j], bx);
      const bool row_emit = (sg >= it.ya && sg < it.yb);   // uniform
      if (!row_emit) continue;
      float4 ic = make_float4(0.f, 0.f, 0.f, 0.f);
      if (col_in) ic = ldg4(a.inv_cnt + (long long)sg * a.Dx + x);
      const int wd = wrap_add(wD, j, DD);
      const int sd = wrap_add(wd, DD - KBG, DD);
      const float4 d4 = ld4(ringD + sd * CW + 4 * tid);
      const float dv[4] = {d4.x, d4.y, d4.z, d4.w};
      const float sv[4] = {bx[0] * ic.x, bx[1] * ic.y, bx[2] * ic.z, bx[3] * ic.w};
      unsigned pass = 0;
#ifdef LPF_DEBUG_FUSED
      if (p == 0 && sg == 20 && x == 36)
        printf("dbg sg=%d x=%d d=%g %g %g %g  s=%g %g %g %g ic=%g bx=%g V2=%g f(sigma)=%g wF=%d wD=%d\n", sg, x, dv[0], dv[1], dv[2], dv[3],
               sv[0], sv[1], sv[2], sv[3], ic.y, bx[1], V2[1], ringF[wrap_add(wrap_add(wF, j, DF), DF - 2 * KBG, DF) * CW + (x + 1 - it.xs)], wF, wD);
#endif
#pragma unroll
      for (int k = 0; k < 4; ++k)
        if (dv[k] > 0.f && dv[k] * dv[k] > a.kappa2 * sv[k] && (x + k) >= it.ux0 && (x + k) < it.ux1) pass |= (1u << k);
      if (pass) {   // rare: guard, local maximum, record
        const int ws = wrap_add(wF, j, DF);
        for (int k = 0; k < 4; ++k) {
          if (!(pass & (1u << k))) continue;
          const int xx = x + k;
          const float d = dv[k];
          const int fs = wrap_add(ws, DF - 2 * KBG, DF);
          const float fv = ringF[fs * CW + (xx - it.xs)];
          const float cc = fv - d;
          const float gd = a.eps_rel * fabsf(cc);
          const float se = fmaxf(sv[k], gd * gd);
          if (!(d * d > a.kappa2 * se)) continue;
          if (!a.W[(long long)sg * a.Dx + xx]) continue;
          bool peak = true;
          for (int dy = -a.k_max; dy <= a.k_max && peak; ++dy) {
            const int yy = sg + dy;
            if (yy < 0 || yy >= a.Dy) continue;
            const int ns = (ws + 2 * DF - 2 * KBG + dy) % DF;
            for (int dx = -a.k_max; dx <= a.k_max; ++dx) {
              const int xn = xx + dx;
              if (xn < 0 || xn >= a.Dx || !a.W[(long long)yy * a.Dx + xn]) continue;
              const int cl = xn - it.xs;
              if (cl < 0 || cl >= CW) continue;
              if (ringF[ns * CW + cl] > fv) { peak = false; break; }
            }
          }
          if (!peak) continue;
          const int idx = atomicAdd(a.ndets, 1);
          if (idx < a.max_det) {
            lpf_det r;
            r.pix = sg * a.Dx + xx; r.plane = (int16_t)p; r.iter = 1;
            r.f = fv; r.c = cc; r.s = se; r.snr = d / sqrtf(se);
            a.dets[idx] = r;
          } else {
            atomicAdd(&a.counters[0], 1);
          }
        }
      }
    }
    wF = wrap_add(wF, RBF, DF);
    wD = wrap_add(wD, RBF, DD);
  }
}

}  // namespace

// ------------------------------------------------------------------------------------------------
// Work plan (host, once per context): column strips over the valid bounding box, row segments.
struct LpfFusedPlan {
  bool ok = false;
  int CW = 0, threads = 0, n_items = 0;
  size_t smem = 0;
  FusedItem* d_items = nullptr;
  float* d_inv_cnt = nullptr;
};

static size_t fused_smem_bytes(int CW) {
  return sizeof(float) * ((size_t)(DF + DD) * CW + RBF * ((CW + 8) + 2 * (CW + 24) + 2 * (CW / 4 + 4)));
}

int lpf_fused_plan(lpf_ctx* c, const uint8_t* hW, LpfFusedPlan** out) {
  *out = nullptr;
  const lpf_params& p = c->p;
  const char* force = getenv("LPF_FORCE_GENERAL");
  if (force && force[0] == '1') return LPF_OK;
  if (!(p.bg_kernel == 1 && p.k_bg == KBG && p.k_mf == 3 && p.sigma_mf > 0 && p.n_iter == 1 && (p.Dx % 4) == 0 && p.k_max <= 2))
    return LPF_OK;
  const int Dy = p.Dy, Dx = p.Dx, H = 2 * KBG + 3;
  // valid bounding box
  int vx0 = Dx, vx1 = 0, vy0 = Dy, vy1 = 0;
  std::vector<int> col_y0(Dx, Dy), col_y1(Dx, 0);
  for (int y = 0; y < Dy; ++y)
    for (int x = 0; x < Dx; ++x)
      if (hW[(size_t)y * Dx + x]) {
        vx0 = std::min(vx0, x); vx1 = std::max(vx1, x + 1); vy0 = std::min(vy0, y); vy1 = std::max(vy1, y + 1);
        col_y0[x] = std::min(col_y0[x], y); col_y1[x] = std::max(col_y1[x], y + 1);
      }
  if (vx1 <= vx0) return LPF_OK;  // nothing valid: general path handles it
  int dev = 0; cudaGetDevice(&dev);
  int max_smem = 0;
  cudaDeviceGetAttribute(&max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
  int cw_max = 4;
  while (cw_max + 4 <= 1024 && fused_smem_bytes(cw_max + 4) <= (size_t)max_smem) cw_max += 4;
  const int width = vx1 - vx0;
  int n_strips = 0, CW = 0;
  std::vector<FusedItem> strips;
  for (int s = 1; s <= 64; ++s) {
    const int uw = ((width + s - 1) / s + 3) / 4 * 4;
    strips.clear();
    int cw = 0;
    for (int i = 0; i < s; ++i) {
      FusedItem it{};
      it.ux0 = vx0 + i * uw; it.ux1 = std::min(vx1, it.ux0 + uw);
      if (it.ux0 >= it.ux1) continue;
      const int lo = std::max(vx0, it.ux0 - H), hi = std::min(vx1, it.ux1 + H);
      it.xs = lo / 4 * 4;
      const int xe = (hi + 3) / 4 * 4;
      cw = std::max(cw, xe - it.xs);
      strips.push_back(it);
    }
    if (cw <= cw_max) { n_strips = (int)strips.size(); CW = cw; break; }
  }
  if (!n_strips) return LPF_OK;
  // row range of each strip and segments: about one CTA per SM per frame
  const int n_planes = c->n_planes;
  const int seg_total = std::max(n_strips, c->n_sm / std::max(1, n_planes));
  std::vector<FusedItem> items;
  long long rows_all = 0;
  for (auto& s : strips) {
    int y0 = Dy, y1 = 0;
    for (int x = s.ux0; x < s.ux1; ++x) { y0 = std::min(y0, col_y0[x]); y1 = std::max(y1, col_y1[x]); }
    s.ya = y0; s.yb = y1;
    rows_all += std::max(0, y1 - y0);
  }
  for (auto& s : strips) {
    const int rows = s.yb - s.ya;
    if (rows <= 0) continue;
    int nseg = (int)std::max<long long>(1, (long long)seg_total * rows / std::max<long long>(1, rows_all));
    nseg = std::min(nseg, std::max(1, rows / 32));
    const int th = (rows + nseg - 1) / nseg;
    for (int k = 0; k < nseg; ++k) {
      FusedItem it = s;
      it.ya = s.ya + k * th; it.yb = std::min(s.yb, it.ya + th);
      if (it.ya < it.yb) items.push_back(it);
    }
  }
  if (items.empty()) return LPF_OK;
  LpfFusedPlan* pl = new LpfFusedPlan();
  pl->CW = CW; pl->threads = CW / 4; pl->n_items = (int)items.size(); pl->smem = fused_smem_bytes(CW);
  if (pl->threads > 256) { delete pl; return LPF_OK; }
  // 1 / (number of valid pixels in the 25x25 window), 0 at invalid pixels: box taps of 1 give exact counts
  LPF_CUDA(cudaMalloc((void**)&pl->d_inv_cnt, (size_t)c->N * sizeof(float)));
  {
    LpfTaps ones;
    ones.R = KBG;
    for (int i = 0; i < LPF_NTAPS; ++i) ones.g[i] = i < WINB ? 1.f : 0.f;
    int rc = lpf_launch_static_norm(c, ones, pl->d_inv_cnt, nullptr, 0);
    if (rc) return rc;
  }
  LPF_CUDA(cudaMalloc((void**)&pl->d_items, items.size() * sizeof(FusedItem)));
  LPF_CUDA(cudaMemcpy(pl->d_items, items.data(), items.size() * sizeof(FusedItem), cudaMemcpyHostToDevice));
  LPF_CUDA(cudaFuncSetAttribute(k_fused_box, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl->smem));
  pl->ok = true;
  *out = pl;
  return LPF_OK;
}

void lpf_fused_plan_free(LpfFusedPlan* pl) {
  if (!pl) return;
  if (pl->d_items) cudaFree(pl->d_items);
  if (pl->d_inv_cnt) cudaFree(pl->d_inv_cnt);
  delete pl;
}

int lpf_fused_plan_info(const LpfFusedPlan* pl, int* cw, int* threads, int* n_items, long long* smem) {
  if (!pl) return 0;
  *cw = pl->CW; *threads = pl->threads; *n_items = pl->n_items; *smem = (long long)pl->smem;
  return 1;
}

int lpf_launch_detect_fused(lpf_ctx* c, LpfFusedPlan* pl, LpfLane& L, const float* d_cube, const uint8_t* d_band_ok,
                            lpf_det* d_dets, int32_t* d_ndets, cudaStream_t st) {
  const lpf_params& p = c->p;
  LPF_CUDA(cudaMemsetAsync(d_ndets, 0, sizeof(int32_t), st));
  if (p.detect_sum_plane) { int rc = lpf_launch_sum_plane(c, L, d_cube, d_band_ok, st); if (rc) return rc; }
  FusedArgs a{};
  a.cube = d_cube; a.sum_plane = L.sum_plane; a.band_ok = d_band_ok; a.W = c->W;
  a.norm_mf = c->norm_mf; a.inv_cnt = pl->d_inv_cnt; a.items = pl->d_items;
  a.B = p.B; a.Dy = p.Dy; a.Dx = p.Dx; a.CW = pl->CW; a.k_max = p.k_max; a.max_det = p.max_det;
  a.g0 = c->g_mf.g[3]; a.g1 = c->g_mf.g[2]; a.g2 = c->g_mf.g[1]; a.g3 = c->g_mf.g[0];
  a.kappa2 = p.kappa * p.kappa; a.eps_rel = p.eps_rel;
  a.dets = d_dets; a.ndets = d_ndets; a.counters = c->counters;
  const dim3 grid(pl->n_items, c->n_planes);
  LPF_KLAUNCH(c, KID_FUSED_DETECT, st, k_fused_box<<<grid, pl->threads, pl->smem, st>>>(a));
  return LPF_OK;
}
