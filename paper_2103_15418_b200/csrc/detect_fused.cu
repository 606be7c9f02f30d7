// S4-S8 fused fast path: matched filter -> local centre -> local spread -> sigma clip -> local
// maxima -> compaction in ONE pass over each plane, for the headline parameter set
// (box background K = 12, Gaussian matched filter k_mf = 3, n_iter = 1).
// (eqs. 2-7; O3-O6 and "Fused detection kernel".)
//
// Design (sm_100a): a CTA owns a column strip (as wide as shared memory allows: the two ring
// buffers of a whole 922-column all-sky strip fill the 227 KB of one SM) and sweeps down a
// segment of rows.  Each thread owns 4 adjacent columns and RBF rows per iteration:
//   A  128-bit global loads of X (masked by W), issued one iteration ahead            [HBM/L2]
//   B  horizontal 7-tap matched filter (neighbour groups through shared memory)
//   C  vertical 7-tap matched filter on a register window, x norm_mf  -> F
//   D  vertical 25-row running sum of F (ring buffer of F rows in shared memory)
//   E  horizontal 25-box of the running sums by blocked partial sums, x 1/count -> C   (eq. 3)
//   F  d = F - C (F re-read from the ring at lag 12)
//   G  vertical 25-row running sum of d^2 (ring buffer of d rows)
//   H  horizontal 25-box, x 1/count                                             -> S   (eq. 4)
//   I  eq. 5 on d at lag 12; pixels that pass take the side path: S_eff guard, eq. 6
//      local-maximum test on the F ring (early exit), eq. 7 record.
// F, C, d and S never leave the SM.  Stages E-G / H-I are skipped while the pipeline warms up
// (27 + 27 rows per segment); no redundant columns when the strip spans the valid width.
#include <algorithm>
#include <cstdio>
#include <cstdlib>

#include "lpf_internal.cuh"

namespace {

constexpr int RBF = 2;         // rows per iteration
constexpr int KBG = 12;        // box half width
constexpr int WINB = 2 * KBG + 1;
constexpr int HALO = 2 * KBG + 3;   // rows of X above the first output row
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
__device__ __forceinline__ float4 zero4() { return make_float4(0.f, 0.f, 0.f, 0.f); }
__device__ __forceinline__ int wrap_add(int a, int b, int m) { const int s = a + b; return s >= m ? s - m : s; }

// horizontal 25-box of one row of per-column values held 4 per thread (group sum of own = t)
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

// Side path for one pixel that passed eq. 5 without the guard: guard (R8), eq. 6 on the F ring, eq. 7.
// Masked pixels hold F = 0 in the ring, so W is consulted only when such a zero would win.
__device__ __noinline__ void fused_candidate(const FusedArgs& a, const FusedItem& it, const float* ringF, int CW,
                                             int slot_sigma, int sg, int xx, float d, float s, int plane) {
  const int cl = xx - it.xs;
  const float fv = ringF[slot_sigma * CW + cl];
  const float cc = fv - d;
  const float gd = a.eps_rel * fabsf(cc);
  const float se = fmaxf(s, gd * gd);
  if (!(d * d > a.kappa2 * se)) return;
  const int km = a.k_max;
  for (int dy = -km; dy <= km; ++dy) {
    const int yy = sg + dy;
    if (yy < 0 || yy >= a.Dy) continue;
    const int ns = (slot_sigma + DF + dy) % DF;
    const float* row = ringF + ns * CW;
    for (int dx = -km; dx <= km; ++dx) {
      const int c2 = cl + dx;
      if (c2 < 0 || c2 >= CW) continue;
      const float fn = row[c2];
      if (fn > fv) {
        const int xn = xx + dx;
        if (xn >= 0 && xn < a.Dx && a.W[(long long)yy * a.Dx + xn]) return;  // a valid neighbour is larger
      }
    }
  }
  const int idx = atomicAdd(a.ndets, 1);
  if (idx < a.max_det) {
    lpf_det r;
    r.pix = sg * a.Dx + xx; r.plane = (int16_t)plane; r.iter = 1;
    r.f = fv; r.c = cc; r.s = se; r.snr = d / sqrtf(se);
    a.dets[idx] = r;
  } else {
    atomicAdd(&a.counters[0], 1);
  }
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
  const int total4 = ((DF + DD) * CW + RBF * (PEX + 2 * PEV + 2 * PET) + 3) >> 2;
  for (int i = tid; i < total4; i += blockDim.x) sm4[i] = zero4();
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

  const int y_start = it.ya - HALO;
  const int nb = (it.yb - it.ya + 2 * HALO + RBF - 1) / RBF;
  // first iteration whose rows reach rho >= ya - KBG (stages E-G) / sigma >= ya (stages H-I)
  const int bE = (HALO + 3 - (RBF - 1)) / RBF;        // rho = y_start + b RBF + j - 15 >= ya - 12
  const int bH = (2 * HALO - (RBF - 1)) / RBF;        // sigma = y_start + b RBF + j - 27 >= ya
  int wF = 0, wD = 0;  // ring slots of the next F row / next d row

  // prefetch of the first rows
  float4 xn[RBF]; unsigned wn[RBF];
#pragma unroll
  for (int j = 0; j < RBF; ++j) {
    const int y = y_start + j;
    xn[j] = zero4(); wn[j] = 0u;
    if (col_in && y >= 0 && y < a.Dy) {
      const long long q = (long long)y * a.Dx + x;
      xn[j] = ldg4(X + q); wn[j] = __ldg(reinterpret_cast<const unsigned*>(a.W + q));
    }
  }

  for (int b = 0; b < nb; ++b) {
    const int yb0 = y_start + b * RBF;
    const bool doE = b >= bE, doH = b >= bH;
    // ---- A: take the prefetched rows, mask, publish; issue this iteration's global loads -----
    float xm[RBF][4];
#pragma unroll
    for (int j = 0; j < RBF; ++j) {
      float4 v = xn[j];
      const unsigned wm = wn[j];
      if (wm != 0x01010101u) {
        if (!(wm & 0x000000ffu)) v.x = 0.f;
        if (!(wm & 0x0000ff00u)) v.y = 0.f;
        if (!(wm & 0x00ff0000u)) v.z = 0.f;
        if (!(wm & 0xff000000u)) v.w = 0.f;
      }
      xm[j][0] = v.x; xm[j][1] = v.y; xm[j][2] = v.z; xm[j][3] = v.w;
      st4(EX + j * PEX + 4 + 4 * tid, v);
    }
    float4 nm[RBF], icr[RBF], ics[RBF];
#pragma unroll
    for (int j = 0; j < RBF; ++j) {
      const int yn = yb0 + RBF + j, fr = yb0 + j - 3, rho = fr - KBG, sg = rho - KBG;
      xn[j] = zero4(); wn[j] = 0u; nm[j] = zero4(); icr[j] = zero4(); ics[j] = zero4();
      if (col_in) {
        if (yn >= 0 && yn < a.Dy && b + 1 < nb) {
          const long long q = (long long)yn * a.Dx + x;
          xn[j] = ldg4(X + q); wn[j] = __ldg(reinterpret_cast<const unsigned*>(a.W + q));
        }
        if (fr >= 0 && fr < a.Dy) nm[j] = ldg4(a.norm_mf + (long long)fr * a.Dx + x);
        if (doE && rho >= 0 && rho < a.Dy) icr[j] = ldg4(a.inv_cnt + (long long)rho * a.Dx + x);
        if (doH && sg >= it.ya && sg < it.yb) ics[j] = ldg4(a.inv_cnt + (long long)sg * a.Dx + x);
      }
    }
    __syncthreads();  // (1)
    // ---- B: horizontal matched filter ----------------------------------------------------
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
      const float nmv[4] = {nm[j].x, nm[j].y, nm[j].z, nm[j].w};
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
      if (doE) {
        st4(EV + j * PEV + 12 + 4 * tid, make_float4(V1[0], V1[1], V1[2], V1[3]));
        t1[j] = (V1[0] + V1[1]) + (V1[2] + V1[3]);
        ET[j * PET + 2 + tid] = t1[j];
      }
    }
    if (doE) {
      __syncthreads();  // (2)
      // ---- E: C = box / count ; F: d = F - C ; G: running sum of d^2 --------------------------
      float t2[RBF];
#pragma unroll
      for (int j = 0; j < RBF; ++j) {
        float bx[4];
        hbox25(EV + j * PEV, ET + j * PET, tid, t1[j], bx);
        const int ws = wrap_add(wF, j, DF);
        const int rs = wrap_add(ws, DF - KBG, DF);
        const float4 fr4 = ld4(ringF + rs * CW + 4 * tid);
        const float d0 = fr4.x - bx[0] * icr[j].x, d1 = fr4.y - bx[1] * icr[j].y;
        const float d2 = fr4.z - bx[2] * icr[j].z, d3 = fr4.w - bx[3] * icr[j].w;
        const int wd = wrap_add(wD, j, DD);
        const int od = wrap_add(wd, DD - WINB, DD);
        const float4 dold = ld4(ringD + od * CW + 4 * tid);
        V2[0] = fmaf(-dold.x, dold.x, fmaf(d0, d0, V2[0]));
        V2[1] = fmaf(-dold.y, dold.y, fmaf(d1, d1, V2[1]));
        V2[2] = fmaf(-dold.z, dold.z, fmaf(d2, d2, V2[2]));
        V2[3] = fmaf(-dold.w, dold.w, fmaf(d3, d3, V2[3]));
        st4(ringD + wd * CW + 4 * tid, make_float4(d0, d1, d2, d3));
        if (doH) {
          st4(EV2 + j * PEV + 12 + 4 * tid, make_float4(V2[0], V2[1], V2[2], V2[3]));
          t2[j] = (V2[0] + V2[1]) + (V2[2] + V2[3]);
          ET2[j * PET + 2 + tid] = t2[j];
        }
      }
      if (doH) {
        __syncthreads();  // (3)
        // ---- H: S = box / count ; I: eq. 5 at sigma = rho - 12 ---------------------------------
#pragma unroll
        for (int j = 0; j < RBF; ++j) {
          const int sg = yb0 + j - 3 - 2 * KBG;
          if (sg < it.ya || sg >= it.yb) continue;   // uniform
          float bx[4];
          hbox25(EV2 + j * PEV, ET2 + j * PET, tid, t2[j], bx);
          const int wd = wrap_add(wD, j, DD);
          const int sd = wrap_add(wd, DD - KBG, DD);
          const float4 d4 = ld4(ringD + sd * CW + 4 * tid);
          const float s0 = bx[0] * ics[j].x, s1 = bx[1] * ics[j].y, s2 = bx[2] * ics[j].z, s3 = bx[3] * ics[j].w;
          const bool p0 = d4.x > 0.f && d4.x * d4.x > a.kappa2 * s0 && x >= it.ux0 && x < it.ux1;
          const bool p1 = d4.y > 0.f && d4.y * d4.y > a.kappa2 * s1 && x + 1 >= it.ux0 && x + 1 < it.ux1;
          const bool p2 = d4.z > 0.f && d4.z * d4.z > a.kappa2 * s2 && x + 2 >= it.ux0 && x + 2 < it.ux1;
          const bool p3 = d4.w > 0.f && d4.w * d4.w > a.kappa2 * s3 && x + 3 >= it.ux0 && x + 3 < it.ux1;
          if (p0 | p1 | p2 | p3) {
            const int slot_sigma = wrap_add(wrap_add(wF, j, DF), DF - 2 * KBG, DF);
            if (p0) fused_candidate(a, it, ringF, CW, slot_sigma, sg, x, d4.x, s0, p);
            if (p1) fused_candidate(a, it, ringF, CW, slot_sigma, sg, x + 1, d4.y, s1, p);
            if (p2) fused_candidate(a, it, ringF, CW, slot_sigma, sg, x + 2, d4.z, s2, p);
            if (p3) fused_candidate(a, it, ringF, CW, slot_sigma, sg, x + 3, d4.w, s3, p);
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
