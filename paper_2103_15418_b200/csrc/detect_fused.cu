// S4-S8 fused fast path: matched filter -> local centre -> local spread -> sigma clip -> local
// maxima -> compaction in ONE pass over each plane, for the headline parameter set
// (box background K = 12, Gaussian matched filter k_mf = 3, n_iter = 1).
// (eqs. 2-7; O3-O6 and "Fused detection kernel".)
//
// Design (sm_100a).  A CTA owns a column strip (4 columns per thread, up to 1024 columns) and sweeps
// down a segment of rows, two rows per iteration, as a three-stage software pipeline with ONE
// block barrier per iteration (the stages of one iteration work on different rows, so their
// shared-memory exchanges are double buffered and independent):
//   A  rows y:        128-bit loads of X two iterations ahead (registers) -> mask -> horizontal
//                     7-tap matched filter with the neighbours' pixels taken by warp shuffles ->
//                     vertical 7-tap on a register window (packed f32x2) -> F(y-3);
//                     25-row running sum V1 += F(y-3) - F(y-28)
//   B  rows rho=y-17: horizontal 25-box of V1 (blocked partial sums) x 1/count -> C (eq. 3);
//                     d = F - C; 25-row running sum V2 += d^2 - d_old^2
//   C  rows sig=y-31: horizontal 25-box of V2 x 1/count -> S (eq. 4); eq. 5 on d(sig); the few
//                     pixels that pass are handed to the whole warp: S_eff guard (R8), eq. 6 on a
//                     32-row shared-memory ring of F with one neighbour per lane, eq. 7 record.
// The 26-row histories of F and d that the running sums and the lagged reads need are private to
// a thread, so they live in TENSOR MEMORY (tcgen05.st/ld 32x32b.x4: 208 of a thread's 256/512
// columns) rather than in shared memory: shared memory carries only what threads exchange.
// Rows x warps that are fully inside the valid region use constant normalisers and load no mask
// or normaliser plane (a per-item class table built by the host plan); F, C, d, S never leave
// the SM.
#include <algorithm>
#include <cstdio>
#include <cstdlib>

#include "lpf_internal.cuh"

namespace {

constexpr int KBG = 12;             // box half width
constexpr int WINB = 2 * KBG + 1;   // 25
constexpr int RB = 2;               // rows per iteration
constexpr int HALO = 2 * KBG + 3;   // rows of X above the first output row (27)
constexpr int LAG_B = 3 + KBG + RB;          // rho = y - 17
constexpr int LAG_C = LAG_B + KBG + RB;      // sig = y - 31
constexpr int DFS = 32;             // shared-memory ring of F rows (local maxima): power of two
constexpr int DT = WINB + 1;        // tensor-memory ring depth (rows) of F and of d
constexpr int TM_D = 4 * DT;        // first tensor-memory column of the d ring (F ring starts at 0)
constexpr int CLS_PAD = 64;         // class table covers rows ya-64 .. yb+64

// class bits of a (row, warp) cell
constexpr int CL_ANYW = 1;   // some valid pixel among the warp's columns +-4
constexpr int CL_ALLW = 2;   // every pixel among the warp's columns +-4 is valid (and in the strip)
constexpr int CL_NM1 = 4;    // norm_mf is the interior constant on all the warp's columns
constexpr int CL_IC1 = 8;    // 1/count is 1/625 on all the warp's columns

struct FusedItem { int xs, ux0, ux1, ya, yb, cls_off, pad0, pad1; };

struct FusedArgs {
  const float* cube; const float* sum_plane; const uint8_t* band_ok; const uint8_t* W;
  const float* norm_mf; const float* inv_cnt; const FusedItem* items; const uint8_t* cls;
  int B, Dy, Dx, CW, k_max, max_det;
  float g0, g1, g2, g3, kappa2, eps_rel, nm_const, ic_const;
  lpf_det* dets; int32_t* ndets; int32_t* counters;
};

__device__ __forceinline__ float4 ld4(const float* p) { return *reinterpret_cast<const float4*>(p); }
__device__ __forceinline__ void st4(float* p, const float4 v) { *reinterpret_cast<float4*>(p) = v; }
__device__ __forceinline__ float4 ldg4(const float* p) { return __ldg(reinterpret_cast<const float4*>(p)); }
__device__ __forceinline__ float4 zero4() { return make_float4(0.f, 0.f, 0.f, 0.f); }

// packed f32x2 arithmetic (FADD2 / FMUL2 / FFMA2: one issue slot for two lanes' worth of fp32)
__device__ __forceinline__ float2 add2(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 mul2(float2 a, float2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ float2 sub2(float2 a, float2 b) { return __ffma2_rn(b, make_float2(-1.f, -1.f), a); }
__device__ __forceinline__ float2 splat(float s) { return make_float2(s, s); }

// ---- tensor memory as a thread-private scratch ring ---------------------------------------------
__device__ __forceinline__ void tm_st4(uint32_t taddr, float2 lo, float2 hi) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};\n"
               ::"r"(taddr), "f"(lo.x), "f"(lo.y), "f"(hi.x), "f"(hi.y) : "memory");
}
__device__ __forceinline__ void tm_ld4(uint32_t taddr, float2& lo, float2& hi) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];\n"
               : "=f"(lo.x), "=f"(lo.y), "=f"(hi.x), "=f"(hi.y) : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tm_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;\n" ::: "memory"); }
__device__ __forceinline__ void tm_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;\n" ::: "memory"); }
// pins a value loaded by tm_ld4 behind the tm_wait_ld that precedes this statement
__device__ __forceinline__ void tm_use(float2& lo, float2& hi) {
  asm volatile("" : "+f"(lo.x), "+f"(lo.y), "+f"(hi.x), "+f"(hi.y));
}

__device__ __forceinline__ int wrap26(int s) { return s >= DT ? s - DT : s; }

__device__ __forceinline__ float4 mask4(float4 v, unsigned wm) {
  if (!(wm & 0x000000ffu)) v.x = 0.f;
  if (!(wm & 0x0000ff00u)) v.y = 0.f;
  if (!(wm & 0x00ff0000u)) v.z = 0.f;
  if (!(wm & 0xff000000u)) v.w = 0.f;
  return v;
}

// horizontal 25-box of a row of per-column values, 4 per thread: the six group sums q-3..q+2 give the
// window of the thread's first column up to one pixel, the other three windows slide.
__device__ __forceinline__ void hbox25(const float* EVrow, const float* ETrow, int tid, float out[4]) {
  const float4 L = ld4(EVrow + 4 * tid);        // group q-3
  const float4 R = ld4(EVrow + 4 * tid + 24);   // group q+3
  const float t0 = ETrow[tid], t1 = ETrow[tid + 1], t2 = ETrow[tid + 2], t3 = ETrow[tid + 3], t4 = ETrow[tid + 4],
              t5 = ETrow[tid + 5];
  out[0] = (((t0 + t1) + (t2 + t3)) + (t4 + t5)) + R.x;
  out[1] = out[0] + (R.y - L.x);
  out[2] = out[1] + (R.z - L.y);
  out[3] = out[2] + (R.w - L.z);
}

struct Prefetch {          // one iteration's worth of input rows, loaded two iterations ahead
  float4 x[RB], xe[RB];    // own 4 pixels; the neighbouring warp's 4 pixels (lanes 0 and 31 only)
  unsigned w[RB], we[RB];  // their mask bytes
};

struct Planes {            // normaliser values of a non-interior cell, loaded one iteration ahead
  float4 nm[RB], icr[RB], ics[RB];
};

template <int NW>
struct Sweep {
  // ---- constants of the thread -----------------------------------------------------------------
  const FusedArgs& a;
  FusedItem it;
  const float* X;
  float* ringF; float* EV1; float* EV2; float* ET1; float* ET2; const uint8_t* cls;
  int tid, lane, warp, x, CW, PEV, PET, plane;
  bool col_in, ld_left, ld_right;
  unsigned umask;
  uint32_t tm;             // tensor-memory address of the thread's column 0
  int y_start;
  // ---- running state -----------------------------------------------------------------------------
  float2 hw[8][2];         // horizontally filtered rows y-7 .. y (rotating, static indices per phase)
  float2 V1[2], V2[2];     // vertical running sums
  Prefetch pf[2];
  Planes pl;
  int w26;                 // tensor-memory ring slot of this iteration's first row

  __device__ __forceinline__ Sweep(const FusedArgs& a_) : a(a_) {}

  __device__ __forceinline__ int cls_at(int row) const { return cls[(row - (it.ya - CLS_PAD)) * NW + warp]; }

  // global loads of the rows y0+j into pf[slot]; rows past y_stop are not needed by any output
  __device__ __forceinline__ void prefetch(int slot, int y0, int y_stop) {
#pragma unroll
    for (int j = 0; j < RB; ++j) {
      const int y = y0 + j;
      Prefetch& p = pf[slot];
      p.x[j] = zero4(); p.xe[j] = zero4(); p.w[j] = 0u; p.we[j] = 0u;
      if (y < 0 || y >= a.Dy || y > y_stop) continue;
      const int c = cls_at(y);
      if (!(c & CL_ANYW)) continue;
      const long long q = (long long)y * a.Dx + x;
      if (c & CL_ALLW) {
        p.w[j] = 0x01010101u; p.we[j] = 0x01010101u;
        if (col_in) p.x[j] = ldg4(X + q);
        if (ld_left) p.xe[j] = ldg4(X + q - 4);
        if (ld_right) p.xe[j] = ldg4(X + q + 4);
      } else {
        if (col_in) { p.x[j] = ldg4(X + q); p.w[j] = __ldg(reinterpret_cast<const unsigned*>(a.W + q)); }
        if (ld_left) { p.xe[j] = ldg4(X + q - 4); p.we[j] = __ldg(reinterpret_cast<const unsigned*>(a.W + q - 4)); }
        if (ld_right) { p.xe[j] = ldg4(X + q + 4); p.we[j] = __ldg(reinterpret_cast<const unsigned*>(a.W + q + 4)); }
      }
    }
  }

  // normaliser planes for the rows the NEXT iteration's stages touch (only where the cell is not interior)
  __device__ __forceinline__ void prefetch_planes(int y0n) {
#pragma unroll
    for (int j = 0; j < RB; ++j) {
      const int fr = y0n + j - 3, rho = y0n + j - LAG_B, sg = y0n + j - LAG_C;
      pl.nm[j] = zero4(); pl.icr[j] = zero4(); pl.ics[j] = zero4();
      if (!col_in) continue;
      if (fr >= 0 && fr < a.Dy && !(cls_at(fr) & CL_NM1)) pl.nm[j] = ldg4(a.norm_mf + (long long)fr * a.Dx + x);
      if (rho >= 0 && rho < a.Dy && !(cls_at(rho) & CL_IC1)) pl.icr[j] = ldg4(a.inv_cnt + (long long)rho * a.Dx + x);
      if (sg >= it.ya && sg < it.yb && !(cls_at(sg) & CL_IC1)) pl.ics[j] = ldg4(a.inv_cnt + (long long)sg * a.Dx + x);
    }
  }

  // eq. 5 guard + eq. 6 + eq. 7 for one pixel that passed the unguarded eq. 5, by the whole warp:
  // lane k < (2 k_max + 1)^2 looks at one neighbour in the shared-memory ring of F.
  __device__ __forceinline__ void candidate(int src, float dsrc, float ssrc, int kcol, int sg) {
    const float d = __shfl_sync(0xffffffffu, dsrc, src);
    const float s = __shfl_sync(0xffffffffu, ssrc, src);
    const int cl = 4 * (warp * 32 + src) + kcol;       // column within the strip
    const float fv = ringF[(sg & (DFS - 1)) * CW + cl];
    const float cc = fv - d;
    const float gd = a.eps_rel * fabsf(cc);
    const float se = fmaxf(s, gd * gd);
    if (!(d > 0.f && d * d > a.kappa2 * se)) return;   // warp-uniform
    const int km = a.k_max, side = 2 * km + 1;
    bool bigger = false;
    if (lane < side * side) {
      const int dy = lane / side - km, dx = lane - (lane / side) * side - km;
      const int yy = sg + dy, c2 = cl + dx, xn = it.xs + c2;
      if (yy >= 0 && yy < a.Dy && c2 >= 0 && c2 < CW && xn < a.Dx) {
        const float fn = ringF[(yy & (DFS - 1)) * CW + c2];
        // masked pixels hold F = 0 in the ring: W is consulted only when such a zero would win
        if (fn > fv) bigger = (fn != 0.f) || (a.W[(long long)yy * a.Dx + xn] != 0);
      }
    }
    if (__any_sync(0xffffffffu, bigger)) return;
    if (lane == 0) {
      const int idx = atomicAdd(a.ndets, 1);
      if (idx < a.max_det) {
        lpf_det r;
        r.pix = sg * a.Dx + it.xs + cl; r.plane = (int16_t)plane; r.iter = 1;
        r.f = fv; r.c = cc; r.s = se; r.snr = d / sqrtf(se);
        a.dets[idx] = r;
      } else {
        atomicAdd(&a.counters[0], 1);
      }
    }
  }

  // One iteration: rows y0, y0+1 enter stage A; PH = iteration index mod 4 fixes the register rotation.
  template <int PH>
  __device__ __forceinline__ void iteration(int b, int nb, int y_stop) {
    const int y0 = y_start + RB * b;
    const int buf = PH & 1, pbuf = buf ^ 1;
    const bool doB = (y0 + 1 - LAG_B) >= it.ya - KBG;     // some rho of this iteration is inside the d range
    const bool doC = (y0 + 1 - LAG_C) >= it.ya;           // some sigma of this iteration is an output row
    const float2 g0 = splat(a.g0), g1 = splat(a.g1), g2 = splat(a.g2), g3 = splat(a.g3);

    // ---- tensor-memory reads of the whole iteration: F(fr-25), F(rho), d(rho-25), d(sig) ------------
    float2 fold[RB][2], flag[RB][2], dold[RB][2], dlag[RB][2];
#pragma unroll
    for (int j = 0; j < RB; ++j) {
      const int so = wrap26(w26 + j + 1), sl = wrap26(w26 + j + KBG);
      tm_ld4(tm + 4 * so, fold[j][0], fold[j][1]);
      tm_ld4(tm + 4 * sl, flag[j][0], flag[j][1]);
      tm_ld4(tm + TM_D + 4 * so, dold[j][0], dold[j][1]);
      tm_ld4(tm + TM_D + 4 * sl, dlag[j][0], dlag[j][1]);
    }

    // ---- stage A, part 1: take the prefetched rows, mask, horizontal matched filter -----------------
    Planes cur = pl;
#pragma unroll
    for (int j = 0; j < RB; ++j) {
      float4 v = pf[buf].x[j], e = pf[buf].xe[j];
      const unsigned wm = pf[buf].w[j], wme = pf[buf].we[j];
      if (wm != 0x01010101u) v = mask4(v, wm);
      if (wme != 0x01010101u) e = mask4(e, wme);
      float l1 = __shfl_up_sync(0xffffffffu, v.y, 1), l2 = __shfl_up_sync(0xffffffffu, v.z, 1),
            l3 = __shfl_up_sync(0xffffffffu, v.w, 1);
      float r0 = __shfl_down_sync(0xffffffffu, v.x, 1), r1 = __shfl_down_sync(0xffffffffu, v.y, 1),
            r2 = __shfl_down_sync(0xffffffffu, v.z, 1);
      if (lane == 0) { l1 = e.y; l2 = e.z; l3 = e.w; }
      if (lane == 31) { r0 = e.x; r1 = e.y; r2 = e.z; }
      const float wv[10] = {l1, l2, l3, v.x, v.y, v.z, v.w, r0, r1, r2};
      float h[4];
#pragma unroll
      for (int k = 0; k < 4; ++k)
        h[k] = fmaf(a.g0, wv[k + 3], fmaf(a.g1, wv[k + 2] + wv[k + 4], fmaf(a.g2, wv[k + 1] + wv[k + 5], a.g3 * (wv[k] + wv[k + 6]))));
      hw[(2 * PH + 6 + j) & 7][0] = make_float2(h[0], h[1]);
      hw[(2 * PH + 6 + j) & 7][1] = make_float2(h[2], h[3]);
    }
    // ---- issue the global loads of iteration b+2 (inputs) and b+1 (normaliser planes) --------------
    prefetch(buf, y0 + 2 * RB, y_stop);
    prefetch_planes(y0 + RB);

    tm_wait_ld();
#pragma unroll
    for (int j = 0; j < RB; ++j) {
      tm_use(fold[j][0], fold[j][1]); tm_use(flag[j][0], flag[j][1]);
      tm_use(dold[j][0], dold[j][1]); tm_use(dlag[j][0], dlag[j][1]);
    }

    // ---- stage A, part 2: vertical matched filter -> F(fr), running sum V1, exchange ----------------
#pragma unroll
    for (int j = 0; j < RB; ++j) {
      const int fr = y0 + j - 3;
      const int cf = (fr >= 0 && fr < a.Dy) ? cls_at(fr) : 0;
      float2 f[2];
#pragma unroll
      for (int p = 0; p < 2; ++p) {
        const float2 h0 = hw[(2 * PH + j + 0) & 7][p], h1 = hw[(2 * PH + j + 1) & 7][p], h2 = hw[(2 * PH + j + 2) & 7][p],
                     h3 = hw[(2 * PH + j + 3) & 7][p], h4 = hw[(2 * PH + j + 4) & 7][p], h5 = hw[(2 * PH + j + 5) & 7][p],
                     h6 = hw[(2 * PH + j + 6) & 7][p];
        f[p] = fma2(g0, h3, fma2(g1, add2(h2, h4), fma2(g2, add2(h1, h5), mul2(g3, add2(h0, h6)))));
      }
      if (fr < it.ya - 2 * KBG) {                      // rows before the segment's first needed F row
        f[0] = splat(0.f); f[1] = splat(0.f);
      } else if (cf & CL_NM1) {
        f[0] = mul2(f[0], splat(a.nm_const)); f[1] = mul2(f[1], splat(a.nm_const));
      } else {
        f[0] = mul2(f[0], make_float2(cur.nm[j].x, cur.nm[j].y)); f[1] = mul2(f[1], make_float2(cur.nm[j].z, cur.nm[j].w));
      }
      V1[0] = add2(V1[0], sub2(f[0], fold[j][0]));
      V1[1] = add2(V1[1], sub2(f[1], fold[j][1]));
      tm_st4(tm + 4 * wrap26(w26 + j), f[0], f[1]);
      st4(ringF + (fr & (DFS - 1)) * CW + 4 * tid, make_float4(f[0].x, f[0].y, f[1].x, f[1].y));
      st4(EV1 + (buf * RB + j) * PEV + KBG + 4 * tid, make_float4(V1[0].x, V1[0].y, V1[1].x, V1[1].y));
      const float2 ts = add2(V1[0], V1[1]);
      ET1[(buf * RB + j) * PET + 3 + tid] = ts.x + ts.y;
    }

    // ---- stage B: C = box(V1) / count at rho ; d = F - C ; running sum V2 of d^2 ---------------------
    if (doB) {
#pragma unroll
      for (int j = 0; j < RB; ++j) {
        const int rho = y0 + j - LAG_B;
        float bx[4];
        hbox25(EV1 + (pbuf * RB + j) * PEV, ET1 + (pbuf * RB + j) * PET, tid, bx);
        const int cr = (rho >= 0 && rho < a.Dy) ? cls_at(rho) : 0;
        float2 ic0, ic1;
        if (rho < it.ya - KBG) { ic0 = splat(0.f); ic1 = splat(0.f); flag[j][0] = splat(0.f); flag[j][1] = splat(0.f); }
        else if (cr & CL_IC1) { ic0 = splat(a.ic_const); ic1 = ic0; }
        else { ic0 = make_float2(cur.icr[j].x, cur.icr[j].y); ic1 = make_float2(cur.icr[j].z, cur.icr[j].w); }
        // d = F - box * (1/count)
        const float2 d0 = fma2(make_float2(-bx[0], -bx[1]), ic0, flag[j][0]);
        const float2 d1 = fma2(make_float2(-bx[2], -bx[3]), ic1, flag[j][1]);
        V2[0] = fma2(make_float2(-dold[j][0].x, -dold[j][0].y), dold[j][0], fma2(d0, d0, V2[0]));
        V2[1] = fma2(make_float2(-dold[j][1].x, -dold[j][1].y), dold[j][1], fma2(d1, d1, V2[1]));
        tm_st4(tm + TM_D + 4 * wrap26(w26 + j), d0, d1);
        st4(EV2 + (buf * RB + j) * PEV + KBG + 4 * tid, make_float4(V2[0].x, V2[0].y, V2[1].x, V2[1].y));
        const float2 ts = add2(V2[0], V2[1]);
        ET2[(buf * RB + j) * PET + 3 + tid] = ts.x + ts.y;
      }
    }

    // ---- stage C: S = box(V2) / count at sigma ; eq. 5 ; candidates -----------------------------------
    if (doC) {
#pragma unroll
      for (int j = 0; j < RB; ++j) {
        const int sg = y0 + j - LAG_C;
        if (sg < it.ya || sg >= it.yb) continue;       // uniform
        float bx[4];
        hbox25(EV2 + (pbuf * RB + j) * PEV, ET2 + (pbuf * RB + j) * PET, tid, bx);
        const int cs = cls_at(sg);
        float2 ic0, ic1;
        if (cs & CL_IC1) { ic0 = splat(a.ic_const); ic1 = ic0; }
        else { ic0 = make_float2(cur.ics[j].x, cur.ics[j].y); ic1 = make_float2(cur.ics[j].z, cur.ics[j].w); }
        const float2 s0 = mul2(make_float2(bx[0], bx[1]), ic0), s1 = mul2(make_float2(bx[2], bx[3]), ic1);
        const float2 k0 = mul2(s0, splat(a.kappa2)), k1 = mul2(s1, splat(a.kappa2));
        const float2 q0 = mul2(dlag[j][0], dlag[j][0]), q1 = mul2(dlag[j][1], dlag[j][1]);
        unsigned bits = (q0.x > k0.x ? 1u : 0u) | (q0.y > k0.y ? 2u : 0u) | (q1.x > k1.x ? 4u : 0u) | (q1.y > k1.y ? 8u : 0u);
        bits &= umask;
        if (__any_sync(0xffffffffu, bits != 0u)) {
          const float dv[4] = {dlag[j][0].x, dlag[j][0].y, dlag[j][1].x, dlag[j][1].y};
          const float sv[4] = {s0.x, s0.y, s1.x, s1.y};
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            unsigned m = __ballot_sync(0xffffffffu, (bits >> k) & 1u);
            while (m) {
              const int src = __ffs(m) - 1;
              m &= m - 1;
              candidate(src, dv[k], sv[k], k, sg);
            }
          }
        }
      }
    }
    w26 = wrap26(w26 + RB);
    (void)nb;
    tm_wait_st();
    __syncthreads();
  }

  __device__ __forceinline__ void run() {
    const int nb = (it.yb - it.ya + HALO + LAG_C + RB - 1) / RB;   // last sigma = yb-1 enters stage C at y = yb-1+LAG_C
    const int y_stop = it.yb - 1 + HALO;                            // last input row any output needs
    prefetch(0, y_start, y_stop);
    prefetch(1, y_start + RB, y_stop);
    prefetch_planes(y_start);
    int b = 0;
    while (true) {
      iteration<0>(b, nb, y_stop); if (++b >= nb) break;
      iteration<1>(b, nb, y_stop); if (++b >= nb) break;
      iteration<2>(b, nb, y_stop); if (++b >= nb) break;
      iteration<3>(b, nb, y_stop); if (++b >= nb) break;
    }
  }
};

template <int NW>
__global__ void __launch_bounds__(NW * 32, 1)
k_fused_box(const FusedArgs a) {
  extern __shared__ float4 sm4[];
  __shared__ uint32_t s_tmem;
  constexpr int TM_COLS = NW > 4 ? 512 : 256;
  float* sm = reinterpret_cast<float*>(sm4);
  const int p = blockIdx.y;
  if (!a.band_ok[a.B]) return;
  if (p < a.B && !a.band_ok[p]) return;

  Sweep<NW> s(a);
  s.it = a.items[blockIdx.x];
  // shared-memory rows are as wide as the CTA (lanes past the strip's CW columns carry zeros)
  s.CW = NW * 128; s.tid = threadIdx.x; s.lane = threadIdx.x & 31; s.warp = threadIdx.x >> 5; s.plane = p;
  s.PEV = s.CW + 2 * KBG; s.PET = NW * 32 + 8;
  s.ringF = sm;
  s.EV1 = s.ringF + DFS * s.CW;
  s.EV2 = s.EV1 + 2 * RB * s.PEV;
  s.ET1 = s.EV2 + 2 * RB * s.PEV;
  s.ET2 = s.ET1 + 2 * RB * s.PET;
  const int nfl = DFS * s.CW + 4 * RB * s.PEV + 4 * RB * s.PET;   // floats, multiple of 4
  uint8_t* cls_s = reinterpret_cast<uint8_t*>(sm + nfl);
  s.cls = cls_s;
  for (int i = s.tid; i < (nfl >> 2); i += NW * 32) sm4[i] = zero4();
  {
    const int nrows = s.it.yb - s.it.ya + 2 * CLS_PAD;
    const uint8_t* src = a.cls + s.it.cls_off;
    for (int i = s.tid; i < nrows * NW; i += NW * 32) cls_s[i] = src[i];
  }
  if (s.warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;\n"
                 ::"l"((uint64_t)__cvta_generic_to_shared(&s_tmem)), "n"(TM_COLS));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n");
  }
  asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
  const uint32_t tm_base = s_tmem;
  // warp w reaches the 32 lanes (w mod 4) * 32 ...; warps w and w+4 share them on different columns
  s.tm = tm_base + ((uint32_t)((s.warp & 3) * 32) << 16) + (uint32_t)(s.warp >> 2) * 256u;
  for (int i = 0; i < 2 * DT; ++i) tm_st4(s.tm + 4 * i, splat(0.f), splat(0.f));
  tm_wait_st();

  const long long N = (long long)a.Dy * a.Dx;
  s.X = (p < a.B) ? a.cube + (long long)p * N : a.sum_plane;
  s.x = s.it.xs + 4 * s.tid;
  s.col_in = 4 * s.tid < a.CW && s.x < a.Dx;
  s.ld_left = s.col_in && s.lane == 0 && s.tid > 0;
  s.ld_right = s.col_in && s.lane == 31 && 4 * (s.tid + 1) < a.CW && s.x + 4 < a.Dx;
  s.umask = 0u;
#pragma unroll
  for (int k = 0; k < 4; ++k)
    if (s.col_in && s.x + k >= s.it.ux0 && s.x + k < s.it.ux1) s.umask |= 1u << k;
  s.y_start = s.it.ya - HALO;
#pragma unroll
  for (int i = 0; i < 8; ++i) { s.hw[i][0] = splat(0.f); s.hw[i][1] = splat(0.f); }
  s.V1[0] = s.V1[1] = s.V2[0] = s.V2[1] = splat(0.f);
  s.w26 = 0;
  __syncthreads();

  s.run();

  tm_wait_st();
  asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
  __syncthreads();
  if (s.warp == 0)
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;\n" ::"r"(tm_base), "n"(TM_COLS));
}

}  // namespace

// ------------------------------------------------------------------------------------------------
// Work plan (host, once per context): column strips over the valid bounding box, row segments,
// and the (row, warp) class table of every strip.
struct LpfFusedPlan {
  bool ok = false;
  int CW = 0, NW = 0, threads = 0, n_items = 0;
  size_t smem = 0;
  float nm_const = 1.f, ic_const = 1.f / 625.f;
  FusedItem* d_items = nullptr;
  uint8_t* d_cls = nullptr;
  float* d_inv_cnt = nullptr;
};

static size_t fused_smem_bytes(int NW, int max_rows) {
  const int CWP = NW * 128, PEV = CWP + 2 * KBG, PET = NW * 32 + 8;
  const size_t nfl = (size_t)DFS * CWP + 4 * RB * PEV + 4 * RB * PET;
  return nfl * sizeof(float) + (((size_t)(max_rows + 2 * CLS_PAD) * NW + 15) & ~(size_t)15);
}

template <int NW>
static cudaError_t fused_launch_t(const FusedArgs& a, dim3 grid, size_t smem, cudaStream_t st, bool set_attr) {
  if (set_attr) return cudaFuncSetAttribute(k_fused_box<NW>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  k_fused_box<NW><<<grid, NW * 32, smem, st>>>(a);
  return cudaSuccess;
}

static cudaError_t fused_dispatch(int NW, const FusedArgs& a, dim3 grid, size_t smem, cudaStream_t st, bool set_attr) {
  switch (NW) {
    case 1: return fused_launch_t<1>(a, grid, smem, st, set_attr);
    case 2: return fused_launch_t<2>(a, grid, smem, st, set_attr);
    case 4: return fused_launch_t<4>(a, grid, smem, st, set_attr);
    default: return fused_launch_t<8>(a, grid, smem, st, set_attr);
  }
}

int lpf_fused_plan(lpf_ctx* c, const uint8_t* hW, LpfFusedPlan** out) {
  *out = nullptr;
  const lpf_params& p = c->p;
  const char* force = getenv("LPF_FORCE_GENERAL");
  if (force && force[0] == '1') return LPF_OK;
  if (!(p.bg_kernel == 1 && p.k_bg == KBG && p.k_mf == 3 && p.sigma_mf > 0 && p.n_iter == 1 && (p.Dx % 4) == 0 && p.k_max <= 2))
    return LPF_OK;
  const int Dy = p.Dy, Dx = p.Dx;
  // valid bounding box, per-column row ranges
  int vx0 = Dx, vx1 = 0, vy0 = Dy, vy1 = 0;
  std::vector<int> col_y0(Dx, Dy), col_y1(Dx, 0);
  for (int y = 0; y < Dy; ++y)
    for (int x = 0; x < Dx; ++x)
      if (hW[(size_t)y * Dx + x]) {
        vx0 = std::min(vx0, x); vx1 = std::max(vx1, x + 1); vy0 = std::min(vy0, y); vy1 = std::max(vy1, y + 1);
        col_y0[x] = std::min(col_y0[x], y); col_y1[x] = std::max(col_y1[x], y + 1);
      }
  if (vx1 <= vx0) return LPF_OK;  // nothing valid: the general path handles it
  // summed-area table of W: counts of valid pixels in (2r+1)^2 windows
  std::vector<int> sat((size_t)(Dy + 1) * (Dx + 1), 0);
  for (int y = 0; y < Dy; ++y) {
    int run = 0;
    for (int x = 0; x < Dx; ++x) {
      run += hW[(size_t)y * Dx + x] ? 1 : 0;
      sat[(size_t)(y + 1) * (Dx + 1) + x + 1] = sat[(size_t)y * (Dx + 1) + x + 1] + run;
    }
  }
  auto full_window = [&](int y, int x, int r) {   // every pixel of the window is in the image and valid
    if (y - r < 0 || x - r < 0 || y + r >= Dy || x + r >= Dx) return false;
    const size_t s = Dx + 1;
    const int n = sat[(size_t)(y + r + 1) * s + x + r + 1] - sat[(size_t)(y - r) * s + x + r + 1] -
                  sat[(size_t)(y + r + 1) * s + x - r] + sat[(size_t)(y - r) * s + x - r];
    return n == (2 * r + 1) * (2 * r + 1);
  };

  // strips: as few as cover the valid width with at most 1024 columns each
  const int width = vx1 - vx0;
  int n_strips = 0, CW = 0;
  std::vector<FusedItem> strips;
  for (int s = 1; s <= 64 && !n_strips; ++s) {
    const int uw = ((width + s - 1) / s + 3) / 4 * 4;
    strips.clear();
    int cw = 0;
    for (int i = 0; i < s; ++i) {
      FusedItem it{};
      it.ux0 = vx0 + i * uw; it.ux1 = std::min(vx1, it.ux0 + uw);
      if (it.ux0 >= it.ux1) continue;
      const int lo = std::max(vx0, it.ux0 - HALO), hi = std::min(vx1, it.ux1 + HALO);
      it.xs = lo / 4 * 4;
      const int xe = std::min(Dx, (hi + 3) / 4 * 4);
      cw = std::max(cw, xe - it.xs);
      strips.push_back(it);
    }
    if (cw <= 1024) { n_strips = (int)strips.size(); CW = cw; }
  }
  if (!n_strips) return LPF_OK;
  int NW = 1;
  while (NW * 128 < CW) NW *= 2;
  // row range of each strip
  long long rows_all = 0;
  for (auto& s : strips) {
    int y0 = Dy, y1 = 0;
    for (int x = s.ux0; x < s.ux1; ++x) { y0 = std::min(y0, col_y0[x]); y1 = std::max(y1, col_y1[x]); }
    s.ya = y0; s.yb = std::max(y0, y1);
    rows_all += s.yb - s.ya;
  }
  if (rows_all <= 0) return LPF_OK;
  // segments per strip: minimise waves x (rows per segment + warm-up cost) over the segment count
  const int n_planes = c->n_planes;
  const double warm = 24.0;   // the 58 warm-up/drain rows of a segment run a part of the pipeline only
  int best_seg = 1; double best_cost = 1e30;
  const int max_rows_strip = (int)(rows_all / n_strips);
  for (int nseg = 1; nseg <= 64; ++nseg) {
    const double rows = (double)max_rows_strip / nseg;
    if (nseg > 1 && rows < 24) break;
    const long long ctas = (long long)nseg * n_strips * n_planes;
    const double waves = (double)((ctas + c->n_sm - 1) / c->n_sm);
    const double cost = waves * (rows + warm);
    if (cost < best_cost - 1e-9) { best_cost = cost; best_seg = nseg; }
  }
  std::vector<FusedItem> items;
  int max_rows = 0;
  for (size_t si = 0; si < strips.size(); ++si) {
    const FusedItem& s = strips[si];
    const int rows = s.yb - s.ya;
    if (rows <= 0) continue;
    const int nseg = std::max(1, std::min(best_seg, rows / 8));
    const int th = (rows + nseg - 1) / nseg;
    for (int k = 0; k < nseg; ++k) {
      FusedItem it = s;
      it.ya = s.ya + k * th; it.yb = std::min(s.yb, it.ya + th);
      it.pad0 = (int)si;
      if (it.ya < it.yb) { items.push_back(it); max_rows = std::max(max_rows, it.yb - it.ya); }
    }
  }
  if (items.empty()) return LPF_OK;
  // class table per item: rows ya-64 .. yb+64, NW cells per row
  std::vector<uint8_t> cls;
  float nm_interior_pix = -1.f;
  long long interior_pix = -1;
  for (auto& it : items) {
    it.cls_off = (int)cls.size();
    const int nrows = it.yb - it.ya + 2 * CLS_PAD;
    cls.resize(cls.size() + (size_t)nrows * NW, 0);
    for (int r = 0; r < nrows; ++r) {
      const int y = it.ya - CLS_PAD + r;
      if (y < 0 || y >= Dy) continue;
      for (int w = 0; w < NW; ++w) {
        const int c0 = it.xs + 128 * w, c1 = std::min(c0 + 128, it.xs + CW);   // own columns [c0, c1)
        if (c0 >= it.xs + CW) continue;
        int any = 0, all = 1, nm1 = 1, ic1 = 1;
        for (int x = c0 - 4; x < c0 + 132; ++x) {
          const bool in = x >= 0 && x < Dx && x >= it.xs - 4 && x < it.xs + CW + 4;
          const bool v = in && hW[(size_t)y * Dx + x];
          any |= v ? 1 : 0;
          if (!v) all = 0;
        }
        if (c1 - c0 < 128) all = 0;   // a partly filled warp takes the guarded path
        for (int x = c0; x < c0 + 128; ++x) {
          if (x >= c1) { nm1 = 0; ic1 = 0; break; }
          if (!full_window(y, x, 3)) nm1 = 0;
          if (!full_window(y, x, KBG)) ic1 = 0;
          if (!nm1 && !ic1) break;
        }
        if (nm1 && interior_pix < 0) interior_pix = (long long)y * Dx + c0;
        cls[(size_t)it.cls_off + (size_t)r * NW + w] =
            (uint8_t)((any ? CL_ANYW : 0) | (all ? CL_ALLW : 0) | (nm1 ? CL_NM1 : 0) | (ic1 ? CL_IC1 : 0));
      }
    }
  }
  (void)nm_interior_pix;
  LpfFusedPlan* pl = new LpfFusedPlan();
  pl->CW = CW; pl->NW = NW; pl->threads = NW * 32; pl->n_items = (int)items.size();
  pl->smem = fused_smem_bytes(NW, max_rows);
  int dev = 0; cudaGetDevice(&dev);
  int max_smem = 0;
  cudaDeviceGetAttribute(&max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
  if (pl->smem > (size_t)max_smem) { delete pl; return LPF_OK; }
  if (interior_pix >= 0) LPF_CUDA(cudaMemcpy(&pl->nm_const, c->norm_mf + interior_pix, sizeof(float), cudaMemcpyDeviceToHost));
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
  LPF_CUDA(cudaMalloc((void**)&pl->d_cls, cls.size()));
  LPF_CUDA(cudaMemcpy(pl->d_cls, cls.data(), cls.size(), cudaMemcpyHostToDevice));
  FusedArgs dummy{};
  LPF_CUDA(fused_dispatch(NW, dummy, dim3(1), pl->smem, 0, true));
  pl->ok = true;
  *out = pl;
  return LPF_OK;
}

void lpf_fused_plan_free(LpfFusedPlan* pl) {
  if (!pl) return;
  if (pl->d_items) cudaFree(pl->d_items);
  if (pl->d_cls) cudaFree(pl->d_cls);
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
  a.norm_mf = c->norm_mf; a.inv_cnt = pl->d_inv_cnt; a.items = pl->d_items; a.cls = pl->d_cls;
  a.B = p.B; a.Dy = p.Dy; a.Dx = p.Dx; a.CW = pl->CW; a.k_max = p.k_max; a.max_det = p.max_det;
  a.g0 = c->g_mf.g[3]; a.g1 = c->g_mf.g[2]; a.g2 = c->g_mf.g[1]; a.g3 = c->g_mf.g[0];
  a.kappa2 = p.kappa * p.kappa; a.eps_rel = p.eps_rel; a.nm_const = pl->nm_const; a.ic_const = pl->ic_const;
  a.dets = d_dets; a.ndets = d_ndets; a.counters = c->counters;
  const dim3 grid(pl->n_items, c->n_planes);
  LPF_KLAUNCH(c, KID_FUSED_DETECT, st, fused_dispatch(pl->NW, a, grid, pl->smem, st, false));
  return LPF_OK;
}
