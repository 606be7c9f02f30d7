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
// Everything a warp has to decide in an iteration (are its input rows all valid / partly masked /
// empty, which normalisers are the interior constants, which stages run) is one 32-bit word of a
// per-item table built by the host plan, so the steady-state iteration is branch-poor and loads
// no mask or normaliser plane inside the valid region.  F, C, d, S never leave the SM.
#include <algorithm>
#include <cstdio>
#include <cstdlib>

#include "lpf_internal.cuh"

extern __shared__ float4 g_sm4[];

namespace {

constexpr int KBG = 12;             // box half width
constexpr int WINB = 2 * KBG + 1;   // 25
constexpr int RB = 2;               // rows per iteration
constexpr int HALO = 2 * KBG + 3;   // rows of X above the first output row (27)
constexpr int LAG_B = 3 + KBG + RB;          // rho = y - 17
constexpr int LAG_C = LAG_B + KBG + RB;      // sig = y - 31
constexpr int DFS = 36;             // shared-memory ring of F rows (local maxima are tested one iteration late)
constexpr int QCAP = 32;            // queued candidates per warp and iteration (more are tested in place)
constexpr int RCAP = 32;            // staged records per warp between flushes
constexpr int DT = WINB + 1;        // tensor-memory ring depth (rows) of F and of d
constexpr int TM_D = 4 * DT;        // first tensor-memory column of the d ring (F ring starts at 0)
constexpr int PADR = 64;            // zero rows above and below the padded normaliser planes

// per-(iteration, warp) control word
constexpr unsigned FL_XMODE = 3u;          // bits 0-1: input rows consumed now: 0 empty, 1 all valid, 2 masked
constexpr int FL_PMODE_SH = 2;             // bits 2-3: the same for the rows loaded now (two iterations ahead)
constexpr unsigned FL_NM_LD = 1u << 4;     // F rows of this iteration use the loaded norm_mf (else the constant)
constexpr unsigned FL_ICR_LD = 1u << 5;    // rho rows use the loaded 1/count
constexpr unsigned FL_ICS_LD = 1u << 6;    // sigma rows use the loaded 1/count
constexpr unsigned FL_NM_PF = 1u << 7;     // load the planes of the next iteration
constexpr unsigned FL_ICR_PF = 1u << 8;
constexpr unsigned FL_ICS_PF = 1u << 9;
constexpr unsigned FL_GATE_A = 1u << 10;   // some F row precedes the segment's first needed one
constexpr unsigned FL_GATE_B = 1u << 11;   // some rho row precedes the segment's first needed one
constexpr unsigned FL_DO_B = 1u << 12;
constexpr unsigned FL_C0 = 1u << 13;       // sigma row j is an output row of this item
constexpr unsigned FL_C1 = 1u << 14;

struct FusedItem { int xs, ux0, ux1, ya, yb, y_start, nb, fl_off; };

struct FusedArgs {
  const float* cube; const float* sum_plane; const uint8_t* band_ok; const uint8_t* W;
  const float* nm_pad; const float* ic_pad;      // [(Dy + 2 PADR)][Dx], zero rows around the image
  const FusedItem* items; const uint32_t* flags;
  int B, Dy, Dx, CW, k_max, max_det;
  float g0, g1, g2, g3, kappa2, eps_rel, nm_const, ic_const;
  lpf_det* dets; int32_t* ndets; int32_t* counters;
};

__device__ __forceinline__ float4 ldg4(const float* p) { return __ldg(reinterpret_cast<const float4*>(p)); }
__device__ __forceinline__ float4 zero4() { return make_float4(0.f, 0.f, 0.f, 0.f); }

// packed f32x2 arithmetic (FADD2 / FMUL2 / FFMA2: one issue slot for two lanes' worth of fp32)
__device__ __forceinline__ float2 add2(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 mul2(float2 a, float2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ float2 sub2(float2 a, float2 b) { return __ffma2_rn(b, make_float2(-1.f, -1.f), a); }
__device__ __forceinline__ float2 splat(float s) { return make_float2(s, s); }
__device__ __forceinline__ float2 neg2(float2 a) { return make_float2(-a.x, -a.y); }

// ---- tensor memory as a thread-private scratch ring ---------------------------------------------
__device__ __forceinline__ void tm_st4(uint32_t taddr, float2 lo, float2 hi) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};\n"
               ::"r"(taddr), "f"(lo.x), "f"(lo.y), "f"(hi.x), "f"(hi.y));
}
__device__ __forceinline__ void tm_ld4(uint32_t taddr, float2& lo, float2& hi) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];\n"
               : "=f"(lo.x), "=f"(lo.y), "=f"(hi.x), "=f"(hi.y) : "r"(taddr));
}
__device__ __forceinline__ void tm_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;\n"); }
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

// shared memory through the kernel's one dynamic array: float index -> value
__device__ __forceinline__ float4 lds4(int i) { return *reinterpret_cast<const float4*>(reinterpret_cast<const float*>(g_sm4) + i); }
__device__ __forceinline__ float lds1(int i) { return reinterpret_cast<const float*>(g_sm4)[i]; }
__device__ __forceinline__ void sts4(int i, float4 v) { *reinterpret_cast<float4*>(reinterpret_cast<float*>(g_sm4) + i) = v; }
__device__ __forceinline__ void sts1(int i, float v) { reinterpret_cast<float*>(g_sm4)[i] = v; }

// horizontal 25-box of a row of per-column values, 4 per thread: the six group sums q-3..q+2 give the
// window of the thread's first column up to one pixel, the other three windows slide.
// ev: float index of the thread's group q-3 in the value row; et: index of group sum q-3.
__device__ __forceinline__ void hbox25(int ev, int et, float out[4]) {
  const float4 L = lds4(ev);        // group q-3
  const float4 R = lds4(ev + 24);   // group q+3
  const float t0 = lds1(et), t1 = lds1(et + 1), t2 = lds1(et + 2), t3 = lds1(et + 3), t4 = lds1(et + 4), t5 = lds1(et + 5);
  out[0] = (((t0 + t1) + (t2 + t3)) + (t4 + t5)) + R.x;
  out[1] = out[0] + (R.y - L.x);
  out[2] = out[1] + (R.z - L.y);
  out[3] = out[2] + (R.w - L.z);
}

// ---- candidate path (out of line: it is the rare part, and it keeps the sweep's code small) -------
struct CandCtx {           // what the out-of-line functions need, by value
  const FusedArgs* ap;     // kernel arguments (shared-memory copy)
  int CWP, xs, plane, lane, ring_y0;
  int o_st;                // float index of the warp's record staging area (RCAP x 8 words)
};

// staged records of a warp -> global list: one atomic for the lot.  Returns the new count (0).
__device__ __noinline__ int cand_flush(const FusedArgs* ap, int o_st, int lane, int nrec) {
  if (nrec <= 0) return 0;
  int base = 0;
  if (lane == 0) base = atomicAdd(ap->ndets, nrec);
  base = __shfl_sync(0xffffffffu, base, 0);
  __syncwarp();
  if (lane < nrec) {
    const uint2* r = reinterpret_cast<const uint2*>(reinterpret_cast<const uint32_t*>(g_sm4) + o_st + lane * 8);
    const int idx = base + lane;
    if (idx < ap->max_det) {
      uint2* dst = reinterpret_cast<uint2*>(ap->dets + idx);
      dst[0] = r[0]; dst[1] = r[1]; dst[2] = r[2];
    } else {
      atomicAdd(&ap->counters[0], 1);
    }
  }
  __syncwarp();
  return 0;
}

// eq. 5 guard + eq. 6 + eq. 7 for one pixel that passed the unguarded eq. 5, by the whole warp:
// lane k < (2 k_max + 1)^2 looks at one neighbour in the shared-memory ring of F (float index 0, row
// pitch CWP, DFS rows, row r in slot (r - ring_y0) mod DFS).  d, s: the pixel's residual and spread;
// cl: its column in the strip; sg: its row.  An accepted record is staged in shared memory; returns the
// warp's new staged count (flushing when the stage is full).
__device__ __forceinline__ int cand_test_body(const CandCtx& c, int nrec, float d, float s, int cl, int sg) {
  const FusedArgs& a = *c.ap;
  const int CWP = c.CWP, lane = c.lane;
  const float fv = lds1((unsigned)(sg - c.ring_y0) % DFS * CWP + cl);
  const float cc = fv - d;
  const float gd = a.eps_rel * fabsf(cc);
  const float se = fmaxf(s, gd * gd);
  if (!(d > 0.f && d * d > a.kappa2 * se)) return nrec;   // warp-uniform
  const int km = a.k_max, side = 2 * km + 1;
  bool bigger = false;
  if (lane < side * side) {
    const int row = side == 5 ? (lane * 13) >> 6 : (side == 3 ? (lane * 11) >> 5 : 0);   // lane / side (k_max <= 2)
    const int dy = row - km, dx = lane - row * side - km;
    const int yy = sg + dy, c2 = cl + dx, xn = c.xs + c2;
    if (yy >= 0 && yy < a.Dy && c2 >= 0 && c2 < CWP && xn < a.Dx) {
      const float fn = lds1((unsigned)(yy - c.ring_y0) % DFS * CWP + c2);
      // masked pixels hold F = 0 in the ring: W is consulted only when such a zero would win
      if (fn > fv) bigger = (fn != 0.f) || (a.W[(long long)yy * a.Dx + xn] != 0);
    }
  }
  if (__any_sync(0xffffffffu, bigger)) return nrec;
  if (lane == 0) {
    uint32_t* r = reinterpret_cast<uint32_t*>(g_sm4) + c.o_st + nrec * 8;
    r[0] = (uint32_t)(sg * a.Dx + c.xs + cl);
    r[1] = (uint32_t)(c.plane & 0xffff) | (1u << 16);        // int16 plane, int16 iter = 1
    r[2] = __float_as_uint(fv); r[3] = __float_as_uint(cc); r[4] = __float_as_uint(se);
    r[5] = __float_as_uint(d / sqrtf(se));
  }
  ++nrec;
  if (nrec == RCAP) nrec = cand_flush(c.ap, c.o_st, lane, nrec);
  return nrec;
}

// entries e = first, first + step, ... < total of the CTA's queue qb (per-warp lists of lengths n_mine
// held by lanes < nw, inclusive prefix pre): the calling warp's share of last iteration's candidates
__device__ __noinline__ int cand_drain(CandCtx c, int nrec, int o_q, int nw, int first, int n_mine, int pre) {
  const int total = __shfl_sync(0xffffffffu, pre, nw - 1);
  for (int e = first; e < total; e += nw) {
    const int owner = __popc(__ballot_sync(0xffffffffu, c.lane < nw && pre <= e));
    const int start = __shfl_sync(0xffffffffu, pre - n_mine, owner);
    const float4 q = lds4(o_q + (owner * QCAP + (e - start)) * 4);
    nrec = cand_test_body(c, nrec, q.z, q.w, __float_as_int(q.x), __float_as_int(q.y));
  }
  return nrec;
}

// a row whose candidates do not fit the queue any more (rare): tested in place
__device__ __noinline__ int cand_row_in_place(CandCtx c, int nrec, unsigned bits, float4 dv, float4 sv, int cl0, int sg) {
  for (int k = 0; k < 4; ++k) {
    unsigned m = __ballot_sync(0xffffffffu, (bits >> k) & 1u);
    const float dk = k == 0 ? dv.x : (k == 1 ? dv.y : (k == 2 ? dv.z : dv.w));
    const float sk = k == 0 ? sv.x : (k == 1 ? sv.y : (k == 2 ? sv.z : sv.w));
    while (m) {
      const int src = __ffs(m) - 1;
      m &= m - 1;
      nrec = cand_test_body(c, nrec, __shfl_sync(0xffffffffu, dk, src), __shfl_sync(0xffffffffu, sk, src),
                            __shfl_sync(0xffffffffu, cl0, src) + k, sg);
    }
  }
  return nrec;
}

struct Prefetch {          // one iteration's worth of input rows, loaded two iterations ahead
  float4 x[RB], xe[RB];    // own 4 pixels; the neighbouring warp's 4 pixels (lanes 0 and 31 only)
  unsigned w[RB], we[RB];  // their mask bytes (masked rows only)
};

struct Planes {            // normaliser values of non-interior cells, loaded one iteration ahead
  float4 nm[RB], icr[RB], ics[RB];
};

template <int NW>
struct Sweep {
  static constexpr int CWP = NW * 128;             // shared-memory row pitch: the CTA's full width
  static constexpr int PEV = CWP + 2 * KBG, PET = NW * 32 + 8;
  static constexpr int O_RING = 0;
  static constexpr int O_EV1 = DFS * CWP;
  static constexpr int O_EV2 = O_EV1 + 2 * RB * PEV;
  static constexpr int O_ET1 = O_EV2 + 2 * RB * PEV;
  static constexpr int O_ET2 = O_ET1 + 2 * RB * PET;
  static constexpr int O_Q = O_ET2 + 2 * RB * PET;    // candidate queues, [2][NW][QCAP] x {col, row, d, s}
  static constexpr int O_QN = O_Q + 2 * NW * QCAP * 4;  // their lengths, [2][NW] (padded to 16 words)
  static constexpr int O_ST = O_QN + 16;                // staged records, [NW][RCAP] x 8 words
  static constexpr int O_FL = O_ST + NW * RCAP * 8;     // control words, [nb][NW]
  // ---- constants of the thread -----------------------------------------------------------------
  const FusedArgs& a;
  const FusedArgs* a_sh;   // the same arguments in shared memory (for the out-of-line candidate path)
  int xs, plane, tid, lane, warp;
  int sx, eoff;            // row stride (0 for lanes outside the strip); offset of the edge lanes' extra load
  bool ld_edge;
  unsigned umask;
  uint32_t tm;             // tensor-memory address of the thread's column 0
  int f_lim, r_lim;        // first needed F row (ya - 24), first needed rho row (ya - 12)
  // ---- running state -----------------------------------------------------------------------------
  const float* xp;         // X at the first row of the next prefetch
  const uint8_t* wp;       // W at the same place
  const float* nmp;        // padded norm_mf at the next iteration's first F row
  const float* icrp;       // padded 1/count at the next iteration's first rho row
  const float* icsp;       // padded 1/count at the next iteration's first sigma row
  int y0;                  // first input row of the current iteration
  int w26;                 // tensor-memory ring slot of this iteration's first row
  int wF;                  // shared-memory ring slot of this iteration's first F row
  int ring_y0;             // the row that sits in slot 0 of the shared-memory ring (mod DFS)
  int qcount, nrec;        // candidates queued in this iteration; records staged by this warp
  float2 hw[8][2];         // horizontally filtered rows (rotating; static indices per phase)
  float2 V1[2], V2[2];     // vertical running sums
  Prefetch pf[2];
  Planes pl[2];

  __device__ __forceinline__ Sweep(const FusedArgs& a_) : a(a_) {}

  __device__ __forceinline__ unsigned ctl(int b) const {
    return reinterpret_cast<const uint32_t*>(g_sm4)[O_FL + b * NW + warp];
  }

  __device__ __forceinline__ CandCtx cand_ctx() const {
    CandCtx c;
    c.ap = a_sh; c.CWP = CWP; c.xs = xs; c.plane = plane; c.lane = lane; c.ring_y0 = ring_y0;
    c.o_st = O_ST + warp * RCAP * 8;
    return c;
  }

  // eq. 6 / eq. 7 for the pixels all warps queued in the previous iteration, dealt round-robin to the warps
  __device__ __forceinline__ void process_queue(int qb) {
    const int n_mine = lane < NW ? reinterpret_cast<const int*>(g_sm4)[O_QN + qb * NW + lane] : 0;
    int pre = n_mine;
#pragma unroll
    for (int o = 1; o < NW; o <<= 1) {
      const int t = __shfl_up_sync(0xffffffffu, pre, o);
      if (lane >= o) pre += t;
    }
    if (__shfl_sync(0xffffffffu, pre, NW - 1) > warp)      // something for this warp
      nrec = cand_drain(cand_ctx(), nrec, O_Q + qb * NW * QCAP * 4, NW, warp, n_mine, pre);
  }

  // global loads of two input rows into pf[slot]; mode 1: all valid, 2: masked (W loaded too)
  __device__ __forceinline__ void load_rows(int slot, unsigned mode) {
    if (mode) {
      Prefetch& p = pf[slot];
      p.x[0] = ldg4(xp); p.x[1] = ldg4(xp + sx);
      if (ld_edge) { p.xe[0] = ldg4(xp + eoff); p.xe[1] = ldg4(xp + sx + eoff); }
      if (mode == 2u) {
        p.w[0] = __ldg(reinterpret_cast<const unsigned*>(wp));
        p.w[1] = __ldg(reinterpret_cast<const unsigned*>(wp + sx));
        if (ld_edge) {
          p.we[0] = __ldg(reinterpret_cast<const unsigned*>(wp + eoff));
          p.we[1] = __ldg(reinterpret_cast<const unsigned*>(wp + sx + eoff));
        }
      }
    }
    xp += RB * sx; wp += RB * sx;
  }

  __device__ __forceinline__ void load_planes(int slot, unsigned fl_nm, unsigned fl_icr, unsigned fl_ics) {
    Planes& q = pl[slot];
    if (fl_nm) { q.nm[0] = ldg4(nmp); q.nm[1] = ldg4(nmp + sx); }
    if (fl_icr) { q.icr[0] = ldg4(icrp); q.icr[1] = ldg4(icrp + sx); }
    if (fl_ics) { q.ics[0] = ldg4(icsp); q.ics[1] = ldg4(icsp + sx); }
    nmp += RB * sx; icrp += RB * sx; icsp += RB * sx;
  }

  // One iteration: rows y0, y0+1 enter stage A; PH = iteration index mod 4 fixes the register rotation.
  template <int PH>
  __device__ __forceinline__ void iteration(int b) {
    constexpr int buf = PH & 1, pbuf = buf ^ 1;
    const unsigned fl = ctl(b);
    const float2 g0 = splat(a.g0), g1 = splat(a.g1), g2 = splat(a.g2), g3 = splat(a.g3);
    process_queue(pbuf);

    // ---- tensor-memory reads, first batch: F(fr - 25) ------------------------------------------------
    float2 fold[RB][2];
#pragma unroll
    for (int j = 0; j < RB; ++j) tm_ld4(tm + 4 * wrap26(w26 + j + 1), fold[j][0], fold[j][1]);

    // ---- stage A, part 1: take the prefetched rows, mask, horizontal matched filter -----------------
    {
      float4 v[RB], e[RB];
      const unsigned mode = fl & FL_XMODE;
      if (mode == 0u) {
#pragma unroll
        for (int j = 0; j < RB; ++j) { v[j] = zero4(); e[j] = zero4(); }
      } else {
#pragma unroll
        for (int j = 0; j < RB; ++j) { v[j] = pf[buf].x[j]; e[j] = pf[buf].xe[j]; }
        if (mode == 2u) {
#pragma unroll
          for (int j = 0; j < RB; ++j) { v[j] = mask4(v[j], pf[buf].w[j]); e[j] = mask4(e[j], pf[buf].we[j]); }
        }
      }
#pragma unroll
      for (int j = 0; j < RB; ++j) {
        float l1 = __shfl_up_sync(0xffffffffu, v[j].y, 1), l2 = __shfl_up_sync(0xffffffffu, v[j].z, 1),
              l3 = __shfl_up_sync(0xffffffffu, v[j].w, 1);
        float r0 = __shfl_down_sync(0xffffffffu, v[j].x, 1), r1 = __shfl_down_sync(0xffffffffu, v[j].y, 1),
              r2 = __shfl_down_sync(0xffffffffu, v[j].z, 1);
        if (lane == 0) { l1 = e[j].y; l2 = e[j].z; l3 = e[j].w; }
        if (lane == 31) { r0 = e[j].x; r1 = e[j].y; r2 = e[j].z; }
        const float wv[10] = {l1, l2, l3, v[j].x, v[j].y, v[j].z, v[j].w, r0, r1, r2};
        float h[4];
#pragma unroll
        for (int k = 0; k < 4; ++k)
          h[k] = fmaf(a.g0, wv[k + 3], fmaf(a.g1, wv[k + 2] + wv[k + 4], fmaf(a.g2, wv[k + 1] + wv[k + 5], a.g3 * (wv[k] + wv[k + 6]))));
        hw[(2 * PH + 6 + j) & 7][0] = make_float2(h[0], h[1]);
        hw[(2 * PH + 6 + j) & 7][1] = make_float2(h[2], h[3]);
      }
    }
    // ---- issue the global loads of iteration b+2 (inputs) and b+1 (normaliser planes) --------------
    load_rows(buf, (fl >> FL_PMODE_SH) & 3u);
    load_planes(pbuf, fl & FL_NM_PF, fl & FL_ICR_PF, fl & FL_ICS_PF);

    tm_wait_ld();
#pragma unroll
    for (int j = 0; j < RB; ++j) tm_use(fold[j][0], fold[j][1]);
    // ---- second batch: F(rho), d(rho - 25), d(sigma) -------------------------------------------------
    float2 flag[RB][2], dold[RB][2], dlag[RB][2];
#pragma unroll
    for (int j = 0; j < RB; ++j) {
      const int so = wrap26(w26 + j + 1), sl = wrap26(w26 + j + KBG);
      tm_ld4(tm + 4 * sl, flag[j][0], flag[j][1]);
      tm_ld4(tm + TM_D + 4 * so, dold[j][0], dold[j][1]);
      tm_ld4(tm + TM_D + 4 * sl, dlag[j][0], dlag[j][1]);
    }

    // ---- stage A, part 2: vertical matched filter -> F(fr), running sum V1, exchange ----------------
    {
      float2 f[RB][2];
#pragma unroll
      for (int j = 0; j < RB; ++j)
#pragma unroll
        for (int p = 0; p < 2; ++p) {
          const float2 h0 = hw[(2 * PH + j + 0) & 7][p], h1 = hw[(2 * PH + j + 1) & 7][p], h2 = hw[(2 * PH + j + 2) & 7][p],
                       h3 = hw[(2 * PH + j + 3) & 7][p], h4 = hw[(2 * PH + j + 4) & 7][p], h5 = hw[(2 * PH + j + 5) & 7][p],
                       h6 = hw[(2 * PH + j + 6) & 7][p];
          f[j][p] = fma2(g0, h3, fma2(g1, add2(h2, h4), fma2(g2, add2(h1, h5), mul2(g3, add2(h0, h6)))));
        }
      if (fl & FL_NM_LD) {
#pragma unroll
        for (int j = 0; j < RB; ++j) {
          f[j][0] = mul2(f[j][0], make_float2(pl[buf].nm[j].x, pl[buf].nm[j].y));
          f[j][1] = mul2(f[j][1], make_float2(pl[buf].nm[j].z, pl[buf].nm[j].w));
        }
      } else {
        const float2 c = splat(a.nm_const);
#pragma unroll
        for (int j = 0; j < RB; ++j) { f[j][0] = mul2(f[j][0], c); f[j][1] = mul2(f[j][1], c); }
      }
      if (fl & FL_GATE_A) {                          // rows before the segment's first needed F row
#pragma unroll
        for (int j = 0; j < RB; ++j)
          if (y0 + j - 3 < f_lim) { f[j][0] = splat(0.f); f[j][1] = splat(0.f); }
      }
#pragma unroll
      for (int j = 0; j < RB; ++j) {
        V1[0] = add2(V1[0], sub2(f[j][0], fold[j][0]));
        V1[1] = add2(V1[1], sub2(f[j][1], fold[j][1]));
        tm_st4(tm + 4 * wrap26(w26 + j), f[j][0], f[j][1]);
        sts4(O_RING + (wF + j >= DFS ? wF + j - DFS : wF + j) * CWP + 4 * tid, make_float4(f[j][0].x, f[j][0].y, f[j][1].x, f[j][1].y));
        sts4(O_EV1 + (buf * RB + j) * PEV + KBG + 4 * tid, make_float4(V1[0].x, V1[0].y, V1[1].x, V1[1].y));
        const float2 ts = add2(V1[0], V1[1]);
        sts1(O_ET1 + (buf * RB + j) * PET + 3 + tid, ts.x + ts.y);
      }
    }

    tm_wait_ld();
#pragma unroll
    for (int j = 0; j < RB; ++j) { tm_use(flag[j][0], flag[j][1]); tm_use(dold[j][0], dold[j][1]); tm_use(dlag[j][0], dlag[j][1]); }

    // ---- stage B: C = box(V1) / count at rho ; d = F - C ; running sum V2 of d^2 ---------------------
    if (fl & FL_DO_B) {
      float2 dd[RB][2];
#pragma unroll
      for (int j = 0; j < RB; ++j) {
        float bx[4];
        hbox25(O_EV1 + (pbuf * RB + j) * PEV + 4 * tid, O_ET1 + (pbuf * RB + j) * PET + tid, bx);
        float2 ic0, ic1;
        if (fl & FL_ICR_LD) { ic0 = make_float2(pl[buf].icr[j].x, pl[buf].icr[j].y); ic1 = make_float2(pl[buf].icr[j].z, pl[buf].icr[j].w); }
        else { ic0 = splat(a.ic_const); ic1 = ic0; }
        dd[j][0] = fma2(make_float2(-bx[0], -bx[1]), ic0, flag[j][0]);     // d = F - box * (1/count)
        dd[j][1] = fma2(make_float2(-bx[2], -bx[3]), ic1, flag[j][1]);
      }
      if (fl & FL_GATE_B) {                          // rows before the segment's first needed rho row
#pragma unroll
        for (int j = 0; j < RB; ++j)
          if (y0 + j - LAG_B < r_lim) { dd[j][0] = splat(0.f); dd[j][1] = splat(0.f); }
      }
#pragma unroll
      for (int j = 0; j < RB; ++j) {
        V2[0] = fma2(neg2(dold[j][0]), dold[j][0], fma2(dd[j][0], dd[j][0], V2[0]));
        V2[1] = fma2(neg2(dold[j][1]), dold[j][1], fma2(dd[j][1], dd[j][1], V2[1]));
        tm_st4(tm + TM_D + 4 * wrap26(w26 + j), dd[j][0], dd[j][1]);
        sts4(O_EV2 + (buf * RB + j) * PEV + KBG + 4 * tid, make_float4(V2[0].x, V2[0].y, V2[1].x, V2[1].y));
        const float2 ts = add2(V2[0], V2[1]);
        sts1(O_ET2 + (buf * RB + j) * PET + 3 + tid, ts.x + ts.y);
      }
    }

    // ---- stage C: S = box(V2) / count at sigma ; eq. 5 ; candidates -----------------------------------
    if (fl & (FL_C0 | FL_C1)) {
#pragma unroll
      for (int j = 0; j < RB; ++j) {
        if (!(fl & (FL_C0 << j))) continue;          // uniform
        float bx[4];
        hbox25(O_EV2 + (pbuf * RB + j) * PEV + 4 * tid, O_ET2 + (pbuf * RB + j) * PET + tid, bx);
        float2 ic0, ic1;
        if (fl & FL_ICS_LD) { ic0 = make_float2(pl[buf].ics[j].x, pl[buf].ics[j].y); ic1 = make_float2(pl[buf].ics[j].z, pl[buf].ics[j].w); }
        else { ic0 = splat(a.ic_const); ic1 = ic0; }
        const float2 s0 = mul2(make_float2(bx[0], bx[1]), ic0), s1 = mul2(make_float2(bx[2], bx[3]), ic1);
        const float2 k0 = mul2(s0, splat(a.kappa2)), k1 = mul2(s1, splat(a.kappa2));
        const float2 q0 = mul2(dlag[j][0], dlag[j][0]), q1 = mul2(dlag[j][1], dlag[j][1]);
        unsigned bits = (q0.x > k0.x ? 1u : 0u) | (q0.y > k0.y ? 2u : 0u) | (q1.x > k1.x ? 4u : 0u) | (q1.y > k1.y ? 8u : 0u);
        bits &= umask;
        if (__any_sync(0xffffffffu, bits != 0u)) {
          const float dv[4] = {dlag[j][0].x, dlag[j][0].y, dlag[j][1].x, dlag[j][1].y};
          const float sv[4] = {s0.x, s0.y, s1.x, s1.y};
          const int sg = y0 + j - LAG_C;
          const unsigned lt = (1u << lane) - 1u;
          const int nrow = __popc(__ballot_sync(0xffffffffu, bits & 1u)) + __popc(__ballot_sync(0xffffffffu, bits & 2u)) +
                           __popc(__ballot_sync(0xffffffffu, bits & 4u)) + __popc(__ballot_sync(0xffffffffu, bits & 8u));
          if (qcount + nrow > QCAP) {                // queue full (rare): test the row in place
            nrec = cand_row_in_place(cand_ctx(), nrec, bits, make_float4(dv[0], dv[1], dv[2], dv[3]),
                                     make_float4(sv[0], sv[1], sv[2], sv[3]), 4 * tid, sg);
          } else {
#pragma unroll
            for (int k = 0; k < 4; ++k) {
              const bool on = (bits >> k) & 1u;
              const unsigned m = __ballot_sync(0xffffffffu, on);
              if (on)
                sts4(O_Q + ((buf * NW + warp) * QCAP + qcount + __popc(m & lt)) * 4,
                     make_float4(__int_as_float(4 * tid + k), __int_as_float(sg), dv[k], sv[k]));
              qcount += __popc(m);
            }
          }
        }
      }
    }
    if (lane == 0) reinterpret_cast<int*>(g_sm4)[O_QN + buf * NW + warp] = qcount;
    qcount = 0;
    wF = wF + RB >= DFS ? wF + RB - DFS : wF + RB;
    w26 = wrap26(w26 + RB);
    y0 += RB;
    tm_wait_st();
    __syncthreads();
  }

  __device__ __forceinline__ void run(int nb) {
    // prologue: the input rows of iterations 0 and 1, the planes of iteration 0
    load_rows(0, ctl(0) & FL_XMODE);
    load_rows(1, nb > 1 ? (ctl(1) & FL_XMODE) : 0u);
    {
      const unsigned f0 = ctl(0);
      load_planes(0, f0 & FL_NM_LD, f0 & FL_ICR_LD, f0 & FL_ICS_LD);
    }
    int b = 0;
    while (true) {
      iteration<0>(b); if (++b >= nb) break;
      iteration<1>(b); if (++b >= nb) break;
      iteration<2>(b); if (++b >= nb) break;
      iteration<3>(b); if (++b >= nb) break;
    }
    process_queue((nb - 1) & 1);     // what the last iteration queued
    nrec = cand_flush(a_sh, O_ST + warp * RCAP * 8, lane, nrec);
  }
};

template <int NW>
__global__ void __launch_bounds__(NW * 32, 1)
k_fused_box(const FusedArgs a) {
  __shared__ uint32_t s_tmem;
  __shared__ FusedArgs s_args;
  constexpr int TM_COLS = NW > 4 ? 512 : 256;
  using SW = Sweep<NW>;
  const int p = blockIdx.y;
  if (!a.band_ok[a.B]) return;
  if (p < a.B && !a.band_ok[p]) return;

  SW s(a);
  const FusedItem it = a.items[blockIdx.x];
  s.a_sh = &s_args;
  s.tid = threadIdx.x; s.lane = threadIdx.x & 31; s.warp = threadIdx.x >> 5; s.plane = p; s.xs = it.xs;
  if (s.tid == 0) s_args = a;
  for (int i = s.tid; i < (SW::O_FL >> 2); i += NW * 32) g_sm4[i] = zero4();
  {
    uint32_t* fl_s = reinterpret_cast<uint32_t*>(g_sm4) + SW::O_FL;
    const uint32_t* src = a.flags + it.fl_off;
    for (int i = s.tid; i < it.nb * NW; i += NW * 32) fl_s[i] = src[i];
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
  const float* X = (p < a.B) ? a.cube + (long long)p * N : a.sum_plane;
  const int x = it.xs + 4 * s.tid;
  const bool col_in = 4 * s.tid < a.CW && x < a.Dx;
  const bool ld_left = col_in && s.lane == 0 && s.tid > 0;
  const bool ld_right = col_in && s.lane == 31 && 4 * (s.tid + 1) < a.CW && x + 4 < a.Dx;
  s.ld_edge = ld_left || ld_right;
  s.eoff = ld_left ? -4 : 4;
  s.umask = 0u;
#pragma unroll
  for (int k = 0; k < 4; ++k)
    if (col_in && x + k >= it.ux0 && x + k < it.ux1) s.umask |= 1u << k;
  s.f_lim = it.ya - 2 * KBG; s.r_lim = it.ya - KBG;
  s.y0 = it.y_start;
  if (col_in) {
    s.sx = a.Dx;
    s.xp = X + (long long)it.y_start * a.Dx + x;
    s.wp = a.W + (long long)it.y_start * a.Dx + x;
    s.nmp = a.nm_pad + (long long)(it.y_start - 3 + PADR) * a.Dx + x;
    s.icrp = a.ic_pad + (long long)(it.y_start - LAG_B + PADR) * a.Dx + x;
    s.icsp = a.ic_pad + (long long)(it.y_start - LAG_C + PADR) * a.Dx + x;
  } else {              // lanes outside the strip read the zero row of a padded plane, over and over
    s.sx = 0;
    s.xp = a.nm_pad; s.wp = reinterpret_cast<const uint8_t*>(a.nm_pad);
    s.nmp = a.nm_pad; s.icrp = a.nm_pad; s.icsp = a.nm_pad;
  }
#pragma unroll
  for (int i = 0; i < 8; ++i) { s.hw[i][0] = splat(0.f); s.hw[i][1] = splat(0.f); }
  s.V1[0] = s.V1[1] = s.V2[0] = s.V2[1] = splat(0.f);
#pragma unroll
  for (int q = 0; q < 2; ++q)
#pragma unroll
    for (int j = 0; j < RB; ++j) {
      s.pf[q].x[j] = zero4(); s.pf[q].xe[j] = zero4(); s.pf[q].w[j] = 0u; s.pf[q].we[j] = 0u;
      s.pl[q].nm[j] = zero4(); s.pl[q].icr[j] = zero4(); s.pl[q].ics[j] = zero4();
    }
  s.w26 = 0; s.wF = 0; s.ring_y0 = it.y_start - 3; s.qcount = 0; s.nrec = 0;
  __syncthreads();

  s.run(it.nb);

  tm_wait_st();
  asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
  __syncthreads();
  if (s.warp == 0)
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;\n" ::"r"(tm_base), "n"(TM_COLS));
}

}  // namespace

// ------------------------------------------------------------------------------------------------
// Work plan (host, once per context): column strips over the valid bounding box, row segments,
// the per-(iteration, warp) control words of every item, zero-padded normaliser planes.
struct LpfFusedPlan {
  bool ok = false;
  int CW = 0, NW = 0, threads = 0, n_items = 0;
  size_t smem = 0;
  float nm_const = 1.f, ic_const = 1.f / 625.f;
  FusedItem* d_items = nullptr;
  uint32_t* d_flags = nullptr;
  float* d_nm_pad = nullptr;
  float* d_ic_pad = nullptr;
};

static size_t fused_smem_bytes(int NW, int max_nb) {
  const int CWP = NW * 128, PEV = CWP + 2 * KBG, PET = NW * 32 + 8;
  const size_t nfl = (size_t)DFS * CWP + 4 * RB * PEV + 4 * RB * PET + 2 * NW * QCAP * 4 + 16 + NW * RCAP * 8;
  return (nfl + (size_t)max_nb * NW) * sizeof(float) + 16;
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

// class bits of a (row, warp) cell of a strip
enum { CL_ANYW = 1,    // some valid pixel among the warp's columns +-4
       CL_ALLW = 2,    // every pixel among the warp's columns +-4 is valid (and the warp is full)
       CL_NM1 = 4,     // norm_mf is the interior constant on all the warp's columns
       CL_IC1 = 8 };   // 1/count is 1/625 on all the warp's columns

int lpf_fused_plan(lpf_ctx* c, const uint8_t* hW, LpfFusedPlan** out) {
  *out = nullptr;
  const lpf_params& p = c->p;
  const char* force = getenv("LPF_FORCE_GENERAL");
  if (force && force[0] == '1') return LPF_OK;
  if (!(p.bg_kernel == 1 && p.k_bg == KBG && p.k_mf == 3 && p.sigma_mf > 0 && p.n_iter == 1 && (p.Dx % 4) == 0 &&
        (p.Dy % 2) == 0 && p.k_max <= 2))
    return LPF_OK;
  const int Dy = p.Dy, Dx = p.Dx;
  // valid bounding box, per-column row ranges
  int vx0 = Dx, vx1 = 0;
  std::vector<int> col_y0(Dx, Dy), col_y1(Dx, 0);
  for (int y = 0; y < Dy; ++y)
    for (int x = 0; x < Dx; ++x)
      if (hW[(size_t)y * Dx + x]) {
        vx0 = std::min(vx0, x); vx1 = std::max(vx1, x + 1);
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
    if (rows > 900 && nseg < 64) continue;      // keeps an item's control words within shared memory
    const long long ctas = (long long)nseg * n_strips * n_planes;
    const double waves = (double)((ctas + c->n_sm - 1) / c->n_sm);
    const double cost = waves * (rows + warm);
    if (cost < best_cost - 1e-9) { best_cost = cost; best_seg = nseg; }
  }
  struct ItemEx { FusedItem it; int strip; };
  std::vector<ItemEx> items;
  for (size_t si = 0; si < strips.size(); ++si) {
    const FusedItem& s = strips[si];
    const int rows = s.yb - s.ya;
    if (rows <= 0) continue;
    const int nseg = std::max(1, std::min(best_seg, rows / 8));
    const int th = (rows + nseg - 1) / nseg;
    for (int k = 0; k < nseg; ++k) {
      FusedItem it = s;
      it.ya = s.ya + k * th; it.yb = std::min(s.yb, it.ya + th);
      if (it.ya < it.yb) items.push_back({it, (int)si});
    }
  }
  if (items.empty()) return LPF_OK;
  // (row, warp) classes of every strip, rows -CPAD .. Dy+CPAD
  const int CPAD = 128;
  std::vector<std::vector<uint8_t>> cls(strips.size());
  long long interior_pix = -1;
  for (size_t si = 0; si < strips.size(); ++si) {
    const int xs = strips[si].xs;
    cls[si].assign((size_t)(Dy + 2 * CPAD) * NW, 0);
    for (int y = 0; y < Dy; ++y)
      for (int w = 0; w < NW; ++w) {
        const int c0 = xs + 128 * w, c1 = std::min(c0 + 128, xs + CW);   // own columns [c0, c1)
        if (c0 >= xs + CW) continue;
        int any = 0, all = 1, nm1 = 1, ic1 = 1;
        for (int x = c0 - 4; x < c0 + 132; ++x) {
          const bool in = x >= 0 && x < Dx && x >= xs - 4 && x < xs + CW + 4;
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
        cls[si][(size_t)(y + CPAD) * NW + w] =
            (uint8_t)((any ? CL_ANYW : 0) | (all ? CL_ALLW : 0) | (nm1 ? CL_NM1 : 0) | (ic1 ? CL_IC1 : 0));
      }
  }
  // control words
  std::vector<uint32_t> flags;
  std::vector<FusedItem> ditems;
  int max_nb = 0;
  for (auto& ie : items) {
    FusedItem it = ie.it;
    const std::vector<uint8_t>& cl = cls[ie.strip];
    auto cell = [&](int y, int w) -> int { return (y < -CPAD || y >= Dy + CPAD) ? 0 : cl[(size_t)(y + CPAD) * NW + w]; };
    int ys = it.ya - HALO;
    if (ys & 1) ys -= 1;               // even first row: a row pair never straddles the image edge (Dy is even)
    it.y_start = ys;
    it.nb = (it.yb - 1 + LAG_C - ys) / RB + 1;
    it.fl_off = (int)flags.size();
    max_nb = std::max(max_nb, it.nb);
    auto xmode = [&](int y, int w) -> unsigned {
      const int a0 = cell(y, w), a1 = cell(y + 1, w);
      if (!((a0 | a1) & CL_ANYW)) return 0u;
      return (a0 & a1 & CL_ALLW) ? 1u : 2u;
    };
    auto both = [&](int y, int w, int bit) -> bool { return (cell(y, w) & cell(y + 1, w) & bit) != 0; };
    for (int b = 0; b < it.nb; ++b)
      for (int w = 0; w < NW; ++w) {
        const int y0 = ys + RB * b;
        auto ld_bits = [&](int yy) -> unsigned {
          unsigned f = 0;
          if (!both(yy - 3, w, CL_NM1)) f |= FL_NM_LD;
          if (!both(yy - LAG_B, w, CL_IC1)) f |= FL_ICR_LD;
          const bool c0 = yy - LAG_C >= it.ya && yy - LAG_C < it.yb, c1 = yy + 1 - LAG_C >= it.ya && yy + 1 - LAG_C < it.yb;
          if ((c0 || c1) && !both(yy - LAG_C, w, CL_IC1)) f |= FL_ICS_LD;
          return f;
        };
        unsigned f = xmode(y0, w);
        if (b + 2 < it.nb) f |= xmode(y0 + 2 * RB, w) << FL_PMODE_SH;
        f |= ld_bits(y0);
        if (b + 1 < it.nb) f |= ld_bits(y0 + RB) << 3;     // FL_*_LD -> FL_*_PF
        if (y0 - 3 < it.ya - 2 * KBG) f |= FL_GATE_A;
        if (y0 - LAG_B < it.ya - KBG) f |= FL_GATE_B;
        if (y0 + 1 - LAG_B >= it.ya - KBG) f |= FL_DO_B;
        if (y0 - LAG_C >= it.ya && y0 - LAG_C < it.yb) f |= FL_C0;
        if (y0 + 1 - LAG_C >= it.ya && y0 + 1 - LAG_C < it.yb) f |= FL_C1;
        flags.push_back(f);
      }
    ditems.push_back(it);
  }
  static_assert((FL_NM_LD << 3) == FL_NM_PF && (FL_ICR_LD << 3) == FL_ICR_PF && (FL_ICS_LD << 3) == FL_ICS_PF, "flag layout");

  LpfFusedPlan* pl = new LpfFusedPlan();
  pl->CW = CW; pl->NW = NW; pl->threads = NW * 32; pl->n_items = (int)ditems.size();
  pl->smem = fused_smem_bytes(NW, max_nb);
  int dev = 0; cudaGetDevice(&dev);
  int max_smem = 0;
  cudaDeviceGetAttribute(&max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
  if (pl->smem > (size_t)max_smem) { delete pl; return LPF_OK; }
  *out = pl;   // owned by the context from here on (freed by lpf_destroy on any later failure)
  if (interior_pix >= 0) LPF_CUDA(cudaMemcpy(&pl->nm_const, c->norm_mf + interior_pix, sizeof(float), cudaMemcpyDeviceToHost));
  // zero-padded copies of norm_mf and of 1 / (number of valid pixels in the 25x25 window; 0 at invalid
  // pixels: box taps of 1 give exact counts)
  const size_t npad = (size_t)(Dy + 2 * PADR) * Dx;
  LPF_CUDA(cudaMalloc((void**)&pl->d_nm_pad, npad * sizeof(float)));
  LPF_CUDA(cudaMalloc((void**)&pl->d_ic_pad, npad * sizeof(float)));
  LPF_CUDA(cudaMemset(pl->d_nm_pad, 0, npad * sizeof(float)));
  LPF_CUDA(cudaMemset(pl->d_ic_pad, 0, npad * sizeof(float)));
  LPF_CUDA(cudaMemcpy(pl->d_nm_pad + (size_t)PADR * Dx, c->norm_mf, (size_t)c->N * sizeof(float), cudaMemcpyDeviceToDevice));
  {
    LpfTaps ones;
    ones.R = KBG;
    for (int i = 0; i < LPF_NTAPS; ++i) ones.g[i] = i < WINB ? 1.f : 0.f;
    int rc = lpf_launch_static_norm(c, ones, pl->d_ic_pad + (size_t)PADR * Dx, nullptr, 0);
    if (rc) return rc;
  }
  LPF_CUDA(cudaMalloc((void**)&pl->d_items, ditems.size() * sizeof(FusedItem)));
  LPF_CUDA(cudaMemcpy(pl->d_items, ditems.data(), ditems.size() * sizeof(FusedItem), cudaMemcpyHostToDevice));
  LPF_CUDA(cudaMalloc((void**)&pl->d_flags, flags.size() * sizeof(uint32_t)));
  LPF_CUDA(cudaMemcpy(pl->d_flags, flags.data(), flags.size() * sizeof(uint32_t), cudaMemcpyHostToDevice));
  FusedArgs dummy{};
  LPF_CUDA(fused_dispatch(NW, dummy, dim3(1), pl->smem, 0, true));
  pl->ok = true;
  return LPF_OK;
}

void lpf_fused_plan_free(LpfFusedPlan* pl) {
  if (!pl) return;
  if (pl->d_items) cudaFree(pl->d_items);
  if (pl->d_flags) cudaFree(pl->d_flags);
  if (pl->d_nm_pad) cudaFree(pl->d_nm_pad);
  if (pl->d_ic_pad) cudaFree(pl->d_ic_pad);
  delete pl;
}

int lpf_fused_plan_info(const LpfFusedPlan* pl, int* cw, int* threads, int* n_items, long long* smem) {
  if (!pl || !pl->ok) return 0;
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
  a.nm_pad = pl->d_nm_pad; a.ic_pad = pl->d_ic_pad; a.items = pl->d_items; a.flags = pl->d_flags;
  a.B = p.B; a.Dy = p.Dy; a.Dx = p.Dx; a.CW = pl->CW; a.k_max = p.k_max; a.max_det = p.max_det;
  a.g0 = c->g_mf.g[3]; a.g1 = c->g_mf.g[2]; a.g2 = c->g_mf.g[1]; a.g3 = c->g_mf.g[0];
  a.kappa2 = p.kappa * p.kappa; a.eps_rel = p.eps_rel; a.nm_const = pl->nm_const; a.ic_const = pl->ic_const;
  a.dets = d_dets; a.ndets = d_ndets; a.counters = c->counters;
  const dim3 grid(pl->n_items, c->n_planes);
  LPF_KLAUNCH(c, KID_FUSED_DETECT, st, fused_dispatch(pl->NW, a, grid, pl->smem, st, false));
  return LPF_OK;
}
