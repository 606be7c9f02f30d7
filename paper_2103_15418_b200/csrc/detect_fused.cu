// S4-S8 fused fast path: matched filter -> local centre -> local spread -> sigma clip in ONE pass over
// each plane (k_sweep), local maxima + records in a short follow-up over the few survivors (k_peaks), for
// the headline parameter set (box background K = 12, Gaussian matched filter k_mf = 3, n_iter = 1).
// (eqs. 2-7; O3-O6 and "Fused detection kernel".)
//
// k_sweep (sm_100a).  A CTA owns a column strip (4 columns per thread, 128 per warp) and sweeps down a
// segment of rows, two rows per iteration, as a three-stage software pipeline with ONE block barrier per
// iteration (the stages of one iteration work on different rows, so their shared-memory exchanges are
// double buffered and independent):
//   A  rows y:        the input rows arrive in shared memory by bulk asynchronous copies (TMA,
//                     cp.async.bulk + mbarrier) issued XST - 1 iterations ahead by thread 0; every thread
//                     reads its 4 pixels and both neighbours' with three 128-bit shared loads -> horizontal
//                     7-tap matched filter -> vertical 7-tap on a register window (packed f32x2) -> F(y-3);
//                     25-row running sum V1 += F(y-3) - F(y-28)
//   B  rows rho=y-17: horizontal 25-box of V1 (group sums, every window summed afresh) x 1/count -> C
//                     (eq. 3); d = F - C; 25-row running sum V2 += d^2 - d_old^2
//   C  rows sig=y-31: horizontal 25-box of V2 x 1/count -> S (eq. 4); eq. 5 on d(sig) for the whole row with
//                     four packed operations and one vote; a thread with a hit drops the pixels that a
//                     vertical neighbour of its own columns already beats (F from tensor memory) and appends
//                     one 48-byte entry {pixel, bits, d[4], S[4]} to the CTA's segment of the hit list.
// The 32-row histories of F and d that the running sums and the lagged reads need are private to a
// thread, so they live in TENSOR MEMORY (tcgen05.st/ld 32x32b.x4, two power-of-two rings of 128 columns
// per thread); shared memory carries only what threads exchange and the input stages.  What a warp has to
// decide in an iteration (is there input, which normalisers are the interior constants, which stages run)
// is one 32-bit word of a per-item table built by the host plan.  F, C, d, S never leave the SM.
// A term far above the rest that leaves a running sum leaves the rounding made in its presence behind for the rest
// of the sweep: the sum is then rebuilt from the ring (warp-uniform, rare).  V2 (sums of squares) is rebuilt when it
// has fallen below 1/FAR_RATIO of the largest value it held since it was last exact; V1 (signed) when an F above
// BIG_SIGMA x the plane's rms leaves it (its rounding reaches C divided by 625: only sources of thousands of sigma
// matter there).
// The input is used unmasked when the cube holds exact zeros at every invalid pixel (checked per frame by
// the QC pass); otherwise each thread applies W itself (slow, rare).
//
// k_peaks.  One thread per surviving pixel recomputes F on its (2 k_max + 1)^2 neighbourhood from the raw
// plane with the sweep's own operation order (so the values are the sweep's, bit for bit), applies the
// S_eff guard (R8), the rounded eq. 5, eq. 6 and writes the eq. 7 record.
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
constexpr int DR = 32;              // depth (rows) of the tensor-memory rings of F and d (power of two)
#ifndef LPF_XST
#define LPF_XST 16
#endif
constexpr int XST = LPF_XST;        // input staging stages (iterations in flight, power of two)
constexpr int TM_D = 4 * DR;        // first tensor-memory column of the d ring (F ring starts at 0)
constexpr int PADR = 64;            // zero rows above and below the padded normaliser planes
constexpr float BIG_SIGMA = 64.f;   // V1: "far above the noise" = |F| > BIG_SIGMA x rms of the plane
constexpr float FAR_RATIO = 4096.f; // V2 is rebuilt when it has fallen below 1/FAR_RATIO of the largest value it held since it was last exact:
                                    // the rounding left in a column is ~1e-7 x that value, and a box of 25 columns holds 3-5 such columns,
                                    // so S keeps ~1e-4 relative; ordinary sources (tens of sigma) never get there
constexpr long long HIT_BUDGET = 1ll << 20;   // entries of the hit list of one frame (48 bytes each)
#ifndef LPF_EXP_SKIP
#define LPF_EXP_SKIP 0            // experiment switch (timing only): 1 no stage C, 2 no stage B, 4 no stage A part 2, 8 no stage A part 1
#endif
#ifndef LPF_SWEEP_MAXW
#define LPF_SWEEP_MAXW 1024       // widest column strip of a CTA (1024: 8 warps, 1 CTA per SM; 512: 4 warps, 2 CTAs per SM)
#endif   // "far above the noise": |value| > BIG_SIGMA x rms of the plane

// per-(iteration, warp) control word
constexpr unsigned FL_X = 1u;              // stage A has input: rows in the image, something valid near the warp
constexpr unsigned FL_NM_LD = 1u << 4;     // F rows of this iteration use the loaded norm_mf (else the constant)
constexpr unsigned FL_ICR_LD = 1u << 5;    // rho rows use the loaded 1/count
constexpr unsigned FL_ICS_LD = 1u << 6;    // sigma rows use the loaded 1/count
constexpr unsigned FL_NM_PF = 1u << 7;     // load the planes of the next iteration
constexpr unsigned FL_ICR_PF = 1u << 8;
constexpr unsigned FL_ICS_PF = 1u << 9;
constexpr unsigned FL_DO_B = 1u << 12;
constexpr unsigned FL_C0 = 1u << 13;       // sigma row j is an output row of this item
constexpr unsigned FL_C1 = 1u << 14;

struct FusedItem { int xs, ux0, ux1, ya, yb, y_start, nb, fl_off; };

// one entry of the hit list: the pixels of one thread and row that pass eq. 5 and the vertical pre-filter
struct alignas(16) HitRec { int32_t pix0, bits, pad0, pad1; float d[4]; float s[4]; };

struct FusedArgs {
  const LpfFrameDesc* fd;                        // non-null: cube and dirty_seq come from the frame descriptor
  const float* cube; const float* sum_plane; const uint8_t* band_ok; const uint8_t* W;
  const float* nm_pad; const float* ic_pad;      // [(Dy + 2 PADR)][Dx], zero rows around the image
  const FusedItem* items; const uint32_t* flags;
  const int32_t* dirty; int dirty_seq;           // *dirty == dirty_seq: some invalid pixel of this cube is not an exact zero
  const float* big_thr;                          // [B + 1] BIG_SIGMA x rms of each plane
  int B, Dy, Dx, CW, k_max, max_det, seg_cap, n_items;
  float g0, g1, g2, g3, kappa2, eps_rel, nm_const, ic_const;
  HitRec* hits; int32_t* hit_cnt;                // [segments][seg_cap], [segments]; segment = plane * items + item
  lpf_det* dets; int32_t* ndets; int32_t* counters;
};

__device__ __forceinline__ float4 zero4() { return make_float4(0.f, 0.f, 0.f, 0.f); }
// a global load the compiler may not sink to its use (the normaliser planes are fetched an iteration ahead)
__device__ __forceinline__ float4 ldg4_pinned(const float* p) {
  float4 v;
  asm volatile("ld.global.nc.v4.f32 {%0, %1, %2, %3}, [%4];\n" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
  return v;
}

// packed f32x2 arithmetic (FADD2 / FMUL2 / FFMA2: one issue slot for two lanes' worth of fp32)
__device__ __forceinline__ float2 add2(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 mul2(float2 a, float2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ float2 sub2(float2 a, float2 b) { return __ffma2_rn(b, make_float2(-1.f, -1.f), a); }
__device__ __forceinline__ float2 splat(float s) { return make_float2(s, s); }
__device__ __forceinline__ float2 neg2(float2 a) { return make_float2(-a.x, -a.y); }
__device__ __forceinline__ float amax4(float2 a, float2 b) { return fmaxf(fmaxf(fabsf(a.x), fabsf(a.y)), fmaxf(fabsf(b.x), fabsf(b.y))); }

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

// ---- bulk asynchronous copies (TMA without a tensor map) and their mbarriers ----------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "LPF_WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra LPF_DONE_%=;\n"
      "bra LPF_WAIT_%=;\n"
      "LPF_DONE_%=:\n"
      "}\n" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n"
               ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}

// shared memory through the kernel's one dynamic array: float index -> value
__device__ __forceinline__ float4 lds4(int i) { return *reinterpret_cast<const float4*>(reinterpret_cast<const float*>(g_sm4) + i); }
__device__ __forceinline__ float lds1(int i) { return reinterpret_cast<const float*>(g_sm4)[i]; }
__device__ __forceinline__ void sts4(int i, float4 v) { *reinterpret_cast<float4*>(reinterpret_cast<float*>(g_sm4) + i) = v; }
__device__ __forceinline__ void sts1(int i, float v) { reinterpret_cast<float*>(g_sm4)[i] = v; }

// horizontal 25-box of a row of per-column values, 4 per thread.  The window of the thread's column k is the
// last 4 - k values of group q-3, the groups q-2 .. q+2 (their sums were exchanged) and the first k + 1 values
// of group q+3; every window is summed afresh (no sliding: a huge column that leaves would leave its rounding).
// ev: float index of group q-3 in the value row; et: index of the group sum q-3.
__device__ __forceinline__ void hbox25(int ev, int et, float2& o01, float2& o23) {
  const float4 L = lds4(ev);        // group q-3
  const float4 R = lds4(ev + 24);   // group q+3
  const float t1 = lds1(et + 1), t2 = lds1(et + 2), t3 = lds1(et + 3), t4 = lds1(et + 4), t5 = lds1(et + 5);
  const float a5 = ((t1 + t2) + (t3 + t4)) + t5;
  const float l2 = L.z + L.w, l1 = L.y + l2, l0 = L.x + l1;
  const float r1 = R.x + R.y, r2 = r1 + R.z, r3 = r2 + R.w;
  o01 = add2(add2(make_float2(l0, l1), make_float2(R.x, r1)), splat(a5));
  o23 = add2(add2(make_float2(l2, L.w), make_float2(r2, r3)), splat(a5));
}

// sum over the n ring rows before slot w (rows k = 1 .. n back), of the values (sq = 0) or their squares
__device__ __noinline__ float4 ring_sum(uint32_t ring, int w, int n, int sq) {
  float2 a0 = splat(0.f), a1 = splat(0.f);
  for (int k = 1; k <= n; ++k) {
    float2 lo, hi;
    tm_ld4(ring + 4u * (uint32_t)((w - k) & (DR - 1)), lo, hi);
    tm_wait_ld();
    tm_use(lo, hi);
    if (sq) { a0 = fma2(lo, lo, a0); a1 = fma2(hi, hi, a1); }
    else { a0 = add2(a0, lo); a1 = add2(a1, hi); }
  }
  return make_float4(a0.x, a0.y, a1.x, a1.y);
}

// the slow input path: a cube with something other than an exact zero at an invalid pixel; x0: column of v.l.x
struct Row12 { float4 l, m, r; };
__device__ __noinline__ Row12 mask_row(const FusedArgs* ap, int y, int x0, Row12 v) {
  const FusedArgs& a = *ap;
  float t[12] = {v.l.x, v.l.y, v.l.z, v.l.w, v.m.x, v.m.y, v.m.z, v.m.w, v.r.x, v.r.y, v.r.z, v.r.w};
#pragma unroll
  for (int k = 0; k < 12; ++k) {
    const int x = x0 + k;
    const bool ok = y >= 0 && y < a.Dy && x >= 0 && x < a.Dx && a.W[(long long)y * a.Dx + x] != 0;
    if (!ok) t[k] = 0.f;
  }
  Row12 o;
  o.l = make_float4(t[0], t[1], t[2], t[3]); o.m = make_float4(t[4], t[5], t[6], t[7]); o.r = make_float4(t[8], t[9], t[10], t[11]);
  return o;
}

struct Planes {            // normaliser values of non-interior cells, loaded one iteration ahead
  float4 nm[RB], icr[RB], ics[RB];
};

// the control word of an interior iteration: input, all three stages, every normaliser the interior constant
constexpr unsigned FL_FAST = FL_X | FL_DO_B | FL_C0 | FL_C1;

template <int NW>
struct Sweep {
  static constexpr int NT = NW * 32;
  static constexpr int CWP = NW * 128;             // shared-memory row pitch: the CTA's full width
  static constexpr int XP = CWP + 8;               // staged input row: 4 columns of margin on both sides
  static constexpr int PEV = CWP + 2 * KBG, PET = NW * 32 + 8;
  static constexpr int O_X = 0;
  static constexpr int O_EV1 = O_X + XST * RB * XP;
  static constexpr int O_EV2 = O_EV1 + 2 * RB * PEV;
  static constexpr int O_ET1 = O_EV2 + 2 * RB * PEV;
  static constexpr int O_ET2 = O_ET1 + 2 * RB * PET;
  static constexpr int O_BAR = O_ET2 + 2 * RB * PET;     // XST input barriers + the iteration barrier (8 bytes each)
  static constexpr int O_NH = O_BAR + 2 * XST + 2;       // entries in the CTA's hit segment so far
  static constexpr int O_FL = O_NH + 2;                  // end of the layout
  // ---- constants of the thread -----------------------------------------------------------------
  const FusedArgs& a;
  const FusedArgs* a_sh;   // the same arguments in shared memory (for the out-of-line paths)
  int xs, plane, tid, lane, warp;
  const uint32_t* flp;     // this warp's control words, [nb] with stride NW
  bool col_in, dirty;
  unsigned umask;
  uint32_t tm;             // tensor-memory address of the thread's column 0
  float big2;              // (BIG_SIGMA x rms of the plane)^2: an F above this leaves its rounding in V1
  float2 vmax[2];          // the largest V2 since V2 was last rebuilt from the ring
  bool want_fix2;          // this thread saw V2 fall far below vmax at the end of the last stage B
  HitRec* seg;             // the CTA's segment of the hit list
  const float* nm0;        // padded norm_mf / 1/count at (row 0 of the image, the thread's first column); the zero row
  const float* ic0;        //   of a padded plane for lanes outside the strip (sx = 0)
  int sx;
  // producer (thread 0)
  const float* xrow0;      // X at (y_start, first copied column)
  uint32_t x_dst0;         // shared address of that column in stage 0, row 0
  uint32_t row_bytes;
  int nb, ys;
  // ---- running state -----------------------------------------------------------------------------
  int y0;                  // first input row of the current iteration
  float2 hn[RB][2];        // horizontally filtered input rows of the coming iteration
  float2 acc[6][2];        // vertical matched filter: the partial sums of the next six F rows
  float2 V1[2], V2[2];     // vertical running sums
  Planes pl;               // normalisers of the coming rows (edge cells only)
  // tensor-memory values of the coming iteration, loaded while the CTA sits in the barrier
  float2 fold[RB][2], flag[RB][2], dold[RB][2], dlag[RB][2], fs[4][2];

  __device__ __forceinline__ Sweep(const FusedArgs& a_) : a(a_) {}

  // the control word of iteration b, from global memory (fetched three iterations ahead; 0 past the end)
  __device__ __forceinline__ unsigned ctl(int b) const {
    unsigned v = 0u;
    if (b < nb) asm volatile("ld.global.nc.u32 %0, [%1];\n" : "=r"(v) : "l"(flp + b * NW));
    return v;
  }
  __device__ __forceinline__ uint32_t bar_addr(int stage) const {
    return smem_u32(reinterpret_cast<const float*>(g_sm4) + O_BAR + 2 * stage);
  }

  // the per-iteration barrier of all warps, in two halves (an mbarrier with one arrival per warp)
  __device__ __forceinline__ void sync_arrive() const { __syncwarp(); if (lane == 0) mbar_arrive(bar_addr(XST)); }
  __device__ __forceinline__ void sync_wait(int b) const { mbar_wait(bar_addr(XST), (uint32_t)b & 1u); }

  // thread 0: the two input rows of iteration bb into stage bb mod XST (a plain arrival when they lie outside the image)
  __device__ __forceinline__ void issue_rows(int bb) {
    const int st = bb & (XST - 1);
    const uint32_t bar = bar_addr(st);
    const int y = ys + RB * bb;
    if (bb >= XST) mbar_wait(bar, (uint32_t)((bb / XST) - 1) & 1u);   // its previous phase (complete unless no warp waited for it)
    if (y >= 0 && y + RB <= a.Dy) {
      mbar_expect_tx(bar, RB * row_bytes);
      const float* src = xrow0 + (long long)RB * bb * a.Dx;
      const uint32_t dst = x_dst0 + (uint32_t)(st * RB * XP * 4);
#pragma unroll
      for (int j = 0; j < RB; ++j) bulk_g2s(dst + (uint32_t)(j * XP * 4), src + (long long)j * a.Dx, row_bytes, bar);
    } else {
      mbar_arrive(bar);
    }
  }

  // the normaliser rows of an edge cell; row: first image row wanted
  __device__ __forceinline__ void load_rows(const float* p0, int row, float4 (&dst)[RB]) {
    const float* p = p0 + (long long)(row + PADR) * sx;
#pragma unroll
    for (int j = 0; j < RB; ++j) dst[j] = ldg4_pinned(p + (long long)j * sx);
  }

  // Stage A, part 1 for iteration bn: staged input rows -> horizontal matched filter -> hn.  It touches only the
  // input stages and registers, so it runs in the shadow of the previous iteration's barrier (between the
  // arrival and the wait).  yn: first input row of iteration bn.
  __device__ __forceinline__ void stage_a1(int bn, unsigned fl, int yn) {
    if ((fl & FL_X) && !(LPF_EXP_SKIP & 8)) {
      const int st = bn & (XST - 1);
      mbar_wait(bar_addr(st), (uint32_t)(bn / XST) & 1u);
#pragma unroll
      for (int j = 0; j < RB; ++j) {
        const int xr = O_X + (st * RB + j) * XP + 4 * tid;
        float4 l = lds4(xr), m = lds4(xr + 4), r = lds4(xr + 8);
        if (dirty) {
          Row12 v; v.l = l; v.m = m; v.r = r;
          v = mask_row(a_sh, yn + j, xs + 4 * tid - 4, v);
          l = v.l; m = v.m; r = v.r;
        }
        const float wv[10] = {l.y, l.z, l.w, m.x, m.y, m.z, m.w, r.x, r.y, r.z};
        float h[4];
#pragma unroll
        for (int k = 0; k < 4; ++k)
          h[k] = fmaf(a.g0, wv[k + 3], fmaf(a.g1, wv[k + 2] + wv[k + 4], fmaf(a.g2, wv[k + 1] + wv[k + 5], a.g3 * (wv[k] + wv[k + 6]))));
        hn[j][0] = make_float2(h[0], h[1]);
        hn[j][1] = make_float2(h[2], h[3]);
      }
    } else {
#pragma unroll
      for (int j = 0; j < RB; ++j) { hn[j][0] = splat(0.f); hn[j][1] = splat(0.f); }
    }
  }

  // pixels of the thread's own 3 x 4 block (rows sigma - 1 .. sigma + 1) that some valid neighbour inside the
  // (2 KM + 1)^2 window already beats: F >= 0 and a neighbour above it (a positive F belongs to a valid pixel;
  // a neighbour at 0 may be a masked one, which eq. 6 skips, so nothing is decided against an F < 0 here)
  template <int KM>
  __device__ __forceinline__ unsigned beaten(const float (&fu)[4], const float (&fc)[4], const float (&fd)[4]) const {
    float cm[4], vm[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) { vm[k] = fmaxf(fu[k], fd[k]); cm[k] = fmaxf(vm[k], fc[k]); }
    unsigned out = 0u;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      float e = vm[k];
#pragma unroll
      for (int kk = 0; kk < 4; ++kk)
        if (kk != k && kk - k <= KM && k - kk <= KM) e = fmaxf(e, cm[kk]);
      if (fc[k] >= 0.f && e > fc[k]) out |= 1u << k;
    }
    return out;
  }

  // a thread with eq. 5 hits in sigma row sg: drop what its own block already beats, append the rest as one entry
  __device__ __forceinline__ void emit_hits(unsigned bits, int sg, float2 d0, float2 d1, float2 s0, float2 s1,
                                            float2 fu0, float2 fu1, float2 fc0, float2 fc1, float2 fd0, float2 fd1) {
    if (a.k_max > 0) {
      const float fu[4] = {fu0.x, fu0.y, fu1.x, fu1.y}, fc[4] = {fc0.x, fc0.y, fc1.x, fc1.y}, fd[4] = {fd0.x, fd0.y, fd1.x, fd1.y};
      bits &= ~(a.k_max >= 2 ? beaten<2>(fu, fc, fd) : beaten<1>(fu, fc, fd));
    }
    if (!bits) return;
    const int idx = atomicAdd(reinterpret_cast<int*>(g_sm4) + O_NH, 1);
    if (idx < a.seg_cap) {
      uint4* dst = reinterpret_cast<uint4*>(seg + idx);
      dst[0] = make_uint4((uint32_t)(sg * a.Dx + xs + 4 * tid), bits, 0u, 0u);
      dst[1] = make_uint4(__float_as_uint(d0.x), __float_as_uint(d0.y), __float_as_uint(d1.x), __float_as_uint(d1.y));
      dst[2] = make_uint4(__float_as_uint(s0.x), __float_as_uint(s0.y), __float_as_uint(s1.x), __float_as_uint(s1.y));
    }
  }

  // tensor-memory reads of iteration b: F(fr - 25), F(rho), d(rho - 25), d(sigma), F(sigma - 1 .. sigma + 2).  None of
  // these rows is written in iteration b - 1, so they are issued before that iteration's barrier.
  __device__ __forceinline__ void tm_prefetch(int b) {
    const int w = (RB * b) & (DR - 1);
    auto slot = [&](int k) -> uint32_t { return tm + 4u * (uint32_t)((w + k) & (DR - 1)); };
    const uint32_t t_old0 = slot(7), t_old1 = slot(8);       // rows 25 and 24 back
    const uint32_t t_lag0 = slot(18), t_lag1 = t_lag0 + 4u;  // w + 18 is even: no wrap in between
    tm_ld4(t_old0, fold[0][0], fold[0][1]); tm_ld4(t_old1, fold[1][0], fold[1][1]);
    tm_ld4(t_lag0, flag[0][0], flag[0][1]); tm_ld4(t_lag1, flag[1][0], flag[1][1]);
    tm_ld4(t_old0 + TM_D, dold[0][0], dold[0][1]); tm_ld4(t_old1 + TM_D, dold[1][0], dold[1][1]);
    tm_ld4(t_lag0 + TM_D, dlag[0][0], dlag[0][1]); tm_ld4(t_lag1 + TM_D, dlag[1][0], dlag[1][1]);
#pragma unroll
    for (int k = 0; k < 4; ++k) tm_ld4(slot(3 + k), fs[k][0], fs[k][1]);
  }

  // One iteration: rows y0, y0+1 enter stage A.  fl: this iteration's control word.  FAST: an interior iteration
  // (fl = FL_FAST): no flag is looked at, no normaliser plane is loaded.
  template <bool FAST>
  __device__ __forceinline__ void iteration(int b, unsigned fl, unsigned fl_next, bool fix1, bool fix2) {
    const int buf = b & 1, pbuf = buf ^ 1;
    const float2 g0 = splat(a.g0), g1 = splat(a.g1), g2 = splat(a.g2), g3 = splat(a.g3);
    const int w = (RB * b) & (DR - 1);                       // ring slot of this iteration's first row (even)
    const uint32_t t_new0 = tm + 4u * (uint32_t)w, t_new1 = t_new0 + 4u;

    // ---- stage A, part 2: vertical matched filter -> F(fr), running sum V1, exchange ----------------
    // F(fr) = g3 h(fr-3) + g2 h(fr-2) + g1 h(fr-1) + g0 h(fr) + g1 h(fr+1) + g2 h(fr+2) + g3 h(fr+3), summed in that
    // order: row y adds its term to the six F rows still open and closes F(y - 3) (k_peaks follows the same order)
    if (!(LPF_EXP_SKIP & 4)) {
      float2 f[RB][2];
#pragma unroll
      for (int j = 0; j < RB; ++j)
#pragma unroll
        for (int p = 0; p < 2; ++p) {
          const float2 h = hn[j][p];
          f[j][p] = fma2(g3, h, acc[0][p]);
          acc[0][p] = fma2(g2, h, acc[1][p]);
          acc[1][p] = fma2(g1, h, acc[2][p]);
          acc[2][p] = fma2(g0, h, acc[3][p]);
          acc[3][p] = fma2(g1, h, acc[4][p]);
          acc[4][p] = fma2(g2, h, acc[5][p]);
          acc[5][p] = mul2(g3, h);
        }
      if (!FAST && (fl & FL_NM_LD)) {
#pragma unroll
        for (int j = 0; j < RB; ++j) {
          f[j][0] = mul2(f[j][0], make_float2(pl.nm[j].x, pl.nm[j].y));
          f[j][1] = mul2(f[j][1], make_float2(pl.nm[j].z, pl.nm[j].w));
        }
      } else {
        const float2 c = splat(a.nm_const);
#pragma unroll
        for (int j = 0; j < RB; ++j) { f[j][0] = mul2(f[j][0], c); f[j][1] = mul2(f[j][1], c); }
      }
      float2 v[RB][2];
      if (!FAST && fix1) {
        // something far above the noise leaves the window: rebuild the sums from the ring
        const float4 s23 = ring_sum(tm, w, 23, 0);
        const float2 b0 = make_float2(s23.x, s23.y), b1 = make_float2(s23.z, s23.w);
        v[0][0] = add2(add2(b0, fold[1][0]), f[0][0]); v[0][1] = add2(add2(b1, fold[1][1]), f[0][1]);
        v[1][0] = add2(add2(b0, f[0][0]), f[1][0]);    v[1][1] = add2(add2(b1, f[0][1]), f[1][1]);
      } else {
        v[0][0] = add2(V1[0], sub2(f[0][0], fold[0][0])); v[0][1] = add2(V1[1], sub2(f[0][1], fold[0][1]));
        v[1][0] = add2(v[0][0], sub2(f[1][0], fold[1][0])); v[1][1] = add2(v[0][1], sub2(f[1][1], fold[1][1]));
      }
      V1[0] = v[1][0]; V1[1] = v[1][1];
#pragma unroll
      for (int j = 0; j < RB; ++j) {
        tm_st4(j ? t_new1 : t_new0, f[j][0], f[j][1]);
        sts4(O_EV1 + (buf * RB + j) * PEV + KBG + 4 * tid, make_float4(v[j][0].x, v[j][0].y, v[j][1].x, v[j][1].y));
        const float2 ts = add2(v[j][0], v[j][1]);
        sts1(O_ET1 + (buf * RB + j) * PET + 3 + tid, ts.x + ts.y);
      }
    }
    if (!FAST && (fl & FL_NM_PF)) load_rows(nm0, y0 + RB - 3, pl.nm);           // the next iteration's norm_mf rows

    // ---- stage B: C = box(V1) / count at rho ; d = F - C ; running sum V2 of d^2 ---------------------
    if ((FAST || (fl & FL_DO_B)) && !(LPF_EXP_SKIP & 2)) {
      float2 dd[RB][2];
#pragma unroll
      for (int j = 0; j < RB; ++j) {
        float2 b01, b23;
        hbox25(O_EV1 + (pbuf * RB + j) * PEV + 4 * tid, O_ET1 + (pbuf * RB + j) * PET + tid, b01, b23);
        float2 ic0, ic1;
        if (!FAST && (fl & FL_ICR_LD)) { ic0 = make_float2(pl.icr[j].x, pl.icr[j].y); ic1 = make_float2(pl.icr[j].z, pl.icr[j].w); }
        else { ic0 = splat(a.ic_const); ic1 = ic0; }
        dd[j][0] = fma2(neg2(b01), ic0, flag[j][0]);     // d = F - box * (1/count)
        dd[j][1] = fma2(neg2(b23), ic1, flag[j][1]);
      }
      if (!FAST && fix2) {
        // V2 had fallen far below what it held since it was last exact (seen at the end of the previous iteration):
        // the roundings made in the presence of the large terms are now a visible part of it.  Rebuild it from the
        // ring (the 25 rows up to the previous iteration's last; warp-uniform, rare) before it is used again.
        const float4 s25 = ring_sum(tm + TM_D, w, 25, 1);
        V2[0] = make_float2(s25.x, s25.y); V2[1] = make_float2(s25.z, s25.w);
        vmax[0] = V2[0]; vmax[1] = V2[1];
      }
      float2 v[RB][2];
      v[0][0] = fma2(neg2(dold[0][0]), dold[0][0], fma2(dd[0][0], dd[0][0], V2[0]));
      v[0][1] = fma2(neg2(dold[0][1]), dold[0][1], fma2(dd[0][1], dd[0][1], V2[1]));
      v[1][0] = fma2(neg2(dold[1][0]), dold[1][0], fma2(dd[1][0], dd[1][0], v[0][0]));
      v[1][1] = fma2(neg2(dold[1][1]), dold[1][1], fma2(dd[1][1], dd[1][1], v[0][1]));
      vmax[0] = make_float2(fmaxf(vmax[0].x, v[1][0].x), fmaxf(vmax[0].y, v[1][0].y));
      vmax[1] = make_float2(fmaxf(vmax[1].x, v[1][1].x), fmaxf(vmax[1].y, v[1][1].y));
      V2[0] = v[1][0]; V2[1] = v[1][1];
      {
        // has V2 fallen below 1 / FAR_RATIO of the largest value it held since it was last exact?  Where the sweep
        // leaves the valid region a column's sum falls to (a rounding of) zero, which is no error worth a rebuild:
        // a column counts only while its own pixel of this row is valid (its 1/count is not 0).
        const float2 r = splat(FAR_RATIO);
        float2 e0 = fma2(V2[0], r, neg2(vmax[0])), e1 = fma2(V2[1], r, neg2(vmax[1]));
        if (!FAST && (fl & FL_ICR_LD)) {
          if (pl.icr[1].x == 0.f) e0.x = 0.f;
          if (pl.icr[1].y == 0.f) e0.y = 0.f;
          if (pl.icr[1].z == 0.f) e1.x = 0.f;
          if (pl.icr[1].w == 0.f) e1.y = 0.f;
        }
        want_fix2 = fminf(fminf(e0.x, e0.y), fminf(e1.x, e1.y)) < 0.f;
      }
#pragma unroll
      for (int j = 0; j < RB; ++j) {
        tm_st4((j ? t_new1 : t_new0) + TM_D, dd[j][0], dd[j][1]);
        sts4(O_EV2 + (buf * RB + j) * PEV + KBG + 4 * tid, make_float4(v[j][0].x, v[j][0].y, v[j][1].x, v[j][1].y));
        const float2 ts = add2(v[j][0], v[j][1]);
        sts1(O_ET2 + (buf * RB + j) * PET + 3 + tid, ts.x + ts.y);
      }
    }
    if (!FAST && (fl & FL_ICR_PF)) load_rows(ic0, y0 + RB - LAG_B, pl.icr);

    // ---- stage C: S = box(V2) / count at sigma ; eq. 5 for the row ; hits ------------------------------
    // (both rows' arithmetic first, in one block with stages A2 and B for the instruction scheduler; then the hits)
    if ((FAST || (fl & (FL_C0 | FL_C1))) && !(LPF_EXP_SKIP & 1)) {
      float2 s0[RB], s1[RB], m0[RB], m1[RB];
      float mm[RB];
#pragma unroll
      for (int j = 0; j < RB; ++j) {
        float2 b01, b23;
        hbox25(O_EV2 + (pbuf * RB + j) * PEV + 4 * tid, O_ET2 + (pbuf * RB + j) * PET + tid, b01, b23);
        float2 ic0, ic1;
        if (!FAST && (fl & FL_ICS_LD)) { ic0 = make_float2(pl.ics[j].x, pl.ics[j].y); ic1 = make_float2(pl.ics[j].z, pl.ics[j].w); }
        else { ic0 = splat(a.ic_const); ic1 = ic0; }
        s0[j] = mul2(b01, ic0); s1[j] = mul2(b23, ic1);
        const float2 k0 = mul2(s0[j], splat(a.kappa2)), k1 = mul2(s1[j], splat(a.kappa2));
        // d^2 - kappa^2 S > 0 somewhere in the thread's pixels?  (the sign of the difference is exact; k_peaks
        // applies the guarded, rounded test)
        m0[j] = fma2(dlag[j][0], dlag[j][0], neg2(k0)); m1[j] = fma2(dlag[j][1], dlag[j][1], neg2(k1));
        mm[j] = fmaxf(fmaxf(m0[j].x, m0[j].y), fmaxf(m1[j].x, m1[j].y));
        if (!FAST && !(fl & (FL_C0 << j))) mm[j] = -1.f;      // not an output row of this item
      }
#pragma unroll
      for (int j = 0; j < RB; ++j) {
        if (mm[j] > 0.f) {
          unsigned bits = 0u;
          if (dlag[j][0].x > 0.f && m0[j].x > 0.f) bits |= 1u;
          if (dlag[j][0].y > 0.f && m0[j].y > 0.f) bits |= 2u;
          if (dlag[j][1].x > 0.f && m1[j].x > 0.f) bits |= 4u;
          if (dlag[j][1].y > 0.f && m1[j].y > 0.f) bits |= 8u;
          bits &= umask;
          if (bits)
            emit_hits(bits, y0 + j - LAG_C, dlag[j][0], dlag[j][1], s0[j], s1[j], fs[j][0], fs[j][1], fs[j + 1][0], fs[j + 1][1],
                      fs[j + 2][0], fs[j + 2][1]);
        }
      }
    }
    if (!FAST && (fl & FL_ICS_PF)) load_rows(ic0, y0 + RB - LAG_C, pl.ics);
    y0 += RB;
    tm_prefetch(b + 1);
    // split barrier: arrive, filter the next iteration's input rows while the slower warps finish, wait
    sync_arrive();
    stage_a1(b + 1, fl_next, y0);
    sync_wait(b);
    tm_wait_st();
  }

  __device__ __forceinline__ void run() {
    unsigned f0 = ctl(0), f1 = ctl(1), f2 = ctl(2);
    if (f0 & FL_NM_LD) load_rows(nm0, y0 - 3, pl.nm);
    if (f0 & FL_ICR_LD) load_rows(ic0, y0 - LAG_B, pl.icr);
    if (f0 & FL_ICS_LD) load_rows(ic0, y0 - LAG_C, pl.ics);
    tm_prefetch(0);
    stage_a1(0, f0, y0);
    for (int b = 0; b < nb; ++b) {
      const unsigned f3 = ctl(b + 3);
      tm_wait_ld();
#pragma unroll
      for (int j = 0; j < RB; ++j) { tm_use(fold[j][0], fold[j][1]); tm_use(flag[j][0], flag[j][1]); tm_use(dold[j][0], dold[j][1]); tm_use(dlag[j][0], dlag[j][1]); }
#pragma unroll
      for (int k = 0; k < 4; ++k) tm_use(fs[k][0], fs[k][1]);
      // the two rare repairs of the running sums live in the slow form of the iteration only: the interior form
      // has no call in it
      const float hot = fmaxf(amax4(fold[0][0], fold[0][1]), amax4(fold[1][0], fold[1][1]));
      const bool h1 = hot * hot > big2;
      if (f0 == FL_FAST && !__any_sync(0xffffffffu, h1 || want_fix2)) {
        iteration<true>(b, f0, f1, false, false);
      } else {
        const bool fix1 = __any_sync(0xffffffffu, h1), fix2 = __any_sync(0xffffffffu, want_fix2);
        want_fix2 = false;
        iteration<false>(b, f0, f1, fix1, fix2);
      }
      f0 = f1; f1 = f2; f2 = f3;
    }
    tm_wait_ld();        // the reads issued for an iteration past the end
  }
};

template <int NW>
__global__ void __launch_bounds__(NW * 32 + 32, NW > 4 ? 1 : 2)
k_sweep(const FusedArgs a) {
  __shared__ uint32_t s_tmem;
  __shared__ FusedArgs s_args;
  constexpr int TM_COLS = NW > 4 ? 512 : 256;
  using SW = Sweep<NW>;
  const int p = blockIdx.y;
  const int segi = p * gridDim.x + blockIdx.x;
  if (!a.band_ok[a.B] || (p < a.B && !a.band_ok[p])) {
    if (threadIdx.x == 0) a.hit_cnt[segi] = 0;
    return;
  }

  SW s(a);
  const FusedItem it = a.items[blockIdx.x];
  s.a_sh = &s_args;
  s.tid = threadIdx.x; s.lane = threadIdx.x & 31; s.warp = threadIdx.x >> 5; s.plane = p; s.xs = it.xs;
  s.nb = it.nb; s.ys = it.y_start;
  s.dirty = *a.dirty == (a.fd ? a.fd->seq : a.dirty_seq);
  { const float bg = a.big_thr[p]; s.big2 = bg * bg; }
  s.vmax[0] = s.vmax[1] = splat(0.f);
  s.want_fix2 = false;
  s.seg = a.hits + (long long)segi * a.seg_cap;
  if (s.tid == 0) s_args = a;
  constexpr int NT = SW::NT + 32;           // NW sweep warps + the input warp
  for (int i = s.tid; i < ((SW::O_FL + 3) >> 2); i += NT) g_sm4[i] = zero4();
  const bool sweeper = s.warp < NW;
  s.flp = a.flags + it.fl_off + (sweeper ? s.warp : 0);
  if (s.warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;\n"
                 ::"l"((uint64_t)__cvta_generic_to_shared(&s_tmem)), "n"(TM_COLS));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n");
  }
  asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
  if (s.tid == 0) {
#pragma unroll
    for (int i = 0; i < XST; ++i) mbar_init(s.bar_addr(i), 1);
    mbar_init(s.bar_addr(XST), NW + 1);       // one arrival per sweep warp + the input warp's
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  }
  asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");   // the zero fill above precedes the bulk copies
  const uint32_t tm_base = s_tmem;
  // warp w reaches the 32 lanes (w mod 4) * 32 ...; warps w and w+4 share them on different columns
  s.tm = tm_base + ((uint32_t)((s.warp & 3) * 32) << 16) + (uint32_t)(s.warp >> 2) * 256u;
  if (sweeper) {
    for (int i = 0; i < 2 * DR; ++i) tm_st4(s.tm + 4 * i, splat(0.f), splat(0.f));
    tm_wait_st();
  }

  const long long N = (long long)a.Dy * a.Dx;
  const float* X = (p < a.B) ? (a.fd ? a.fd->cube : a.cube) + (long long)p * N : a.sum_plane;
  const int x = it.xs + 4 * s.tid;
  s.col_in = sweeper && 4 * s.tid < a.CW && x < a.Dx;
  s.umask = 0u;
#pragma unroll
  for (int k = 0; k < 4; ++k)
    if (s.col_in && x + k >= it.ux0 && x + k < it.ux1) s.umask |= 1u << k;
  s.y0 = it.y_start;
  {   // copied columns: the strip with 4 columns of margin, clipped to the image
    const int cx0 = it.xs - 4 > 0 ? it.xs - 4 : 0;
    const int cx1 = it.xs + a.CW + 4 < a.Dx ? it.xs + a.CW + 4 : a.Dx;
    s.row_bytes = (uint32_t)(cx1 - cx0) * 4u;
    s.xrow0 = X + (long long)it.y_start * a.Dx + cx0;
    s.x_dst0 = smem_u32(reinterpret_cast<const float*>(g_sm4) + SW::O_X + (cx0 - (it.xs - 4)));
  }
  if (s.col_in) {
    s.sx = a.Dx;
    s.nm0 = a.nm_pad + x; s.ic0 = a.ic_pad + x;
  } else {              // lanes outside the strip read the zero row of a padded plane, over and over
    s.sx = 0;
    s.nm0 = a.nm_pad; s.ic0 = a.nm_pad;
  }
#pragma unroll
  for (int i = 0; i < 6; ++i) { s.acc[i][0] = splat(0.f); s.acc[i][1] = splat(0.f); }
  s.V1[0] = s.V1[1] = s.V2[0] = s.V2[1] = splat(0.f);
#pragma unroll
  for (int j = 0; j < RB; ++j) { s.pl.nm[j] = zero4(); s.pl.icr[j] = zero4(); s.pl.ics[j] = zero4(); }
  __syncthreads();
  if (sweeper) {
    s.run();
    tm_wait_st();
  } else if (s.lane == 0) {
    // the input warp: one thread keeps the 16-stage ring of input rows full.  It takes part in the iteration barrier
    // (its arrival is always early), so it learns that every sweep warp has read the stage of iteration b the moment
    // the barrier of b completes, and its copies never sit on a sweep warp's path.
    for (int bb = 0; bb < XST && bb < it.nb; ++bb) s.issue_rows(bb);
    for (int b = 0; b < it.nb; ++b) {
      mbar_arrive(s.bar_addr(XST));
      s.sync_wait(b);
      if (b + XST < it.nb) s.issue_rows(b + XST);
    }
    // no bulk copy may be in flight when the CTA leaves
    for (int bb = it.nb > XST ? it.nb - XST : 0; bb < it.nb; ++bb) mbar_wait(s.bar_addr(bb & (XST - 1)), (uint32_t)(bb / XST) & 1u);
  }
  asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
  __syncthreads();
  if (s.tid == 0) {
    const int n = reinterpret_cast<const int*>(g_sm4)[SW::O_NH];
    a.hit_cnt[segi] = n < a.seg_cap ? n : a.seg_cap;
    if (n > a.seg_cap) atomicAdd(&a.counters[0], n - a.seg_cap);
#ifdef LPF_DEBUG_HITS
    atomicAdd(&a.counters[1], n);
#endif
  }
  if (s.warp == 0)
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;\n" ::"r"(tm_base), "n"(TM_COLS));
}

// ---- eq. 6 / eq. 7 on the survivors ------------------------------------------------------------------------------
// One THREAD per surviving pixel (the cheapest form in instructions; the kernel is short on parallelism, not on issue
// slots, and shares the SMs with the other lanes' kernels).  F at the pixels of its (2 KM + 1)^2 neighbourhood is
// recomputed from the plane with the sweep's operation order: horizontal 7 taps as nested fused multiply-adds,
// vertical 7 taps oldest row first, x norm_mf - the values are the sweep's, bit for bit.  X counts as 0 outside the
// image and at invalid pixels (the cube holds exact zeros there, or W is applied when it does not: MASKED).
template <int KM, bool MASKED>
__device__ __forceinline__ bool peak_test(const FusedArgs& a, const float* __restrict__ X, int y, int x, float d, float s,
                                          float& fv, float& cc, float& se) {
  constexpr int NR = 2 * KM + 7, NC = 2 * KM + 1;
  float h[NR][NC];
#pragma unroll
  for (int r = 0; r < NR; ++r) {
    const int yy = y - KM - 3 + r;
    float xv[NC + 6];
#pragma unroll
    for (int c = 0; c < NC + 6; ++c) {
      const int xx = x - KM - 3 + c;
      const bool in = yy >= 0 && yy < a.Dy && xx >= 0 && xx < a.Dx;
      const long long q = (long long)yy * a.Dx + xx;
      xv[c] = (in && (!MASKED || a.W[q] != 0)) ? X[q] : 0.f;
    }
#pragma unroll
    for (int c = 0; c < NC; ++c)
      h[r][c] = fmaf(a.g0, xv[c + 3], fmaf(a.g1, xv[c + 2] + xv[c + 4], fmaf(a.g2, xv[c + 1] + xv[c + 5], a.g3 * (xv[c] + xv[c + 6]))));
  }
  auto F = [&](int dy, int dx) -> float {   // F at (y + dy, x + dx), |dy|, |dx| <= KM; 0 at an invalid pixel (norm_mf = 0)
    const int r = dy + KM, c = dx + KM;
    float v = a.g3 * h[r][c];          // the sweep's order: oldest row first, one fused multiply-add per row
    v = fmaf(a.g2, h[r + 1][c], v); v = fmaf(a.g1, h[r + 2][c], v); v = fmaf(a.g0, h[r + 3][c], v);
    v = fmaf(a.g1, h[r + 4][c], v); v = fmaf(a.g2, h[r + 5][c], v); v = fmaf(a.g3, h[r + 6][c], v);
    return v * a.nm_pad[(long long)(y + dy + PADR) * a.Dx + x + dx];
  };
  fv = F(0, 0);
  cc = fv - d;
  const float gd = a.eps_rel * fabsf(cc);
  se = fmaxf(s, gd * gd);
  if (!(d > 0.f && d * d > a.kappa2 * se)) return false;
  bool bigger = false;
#pragma unroll
  for (int dy = -KM; dy <= KM; ++dy)
#pragma unroll
    for (int dx = -KM; dx <= KM; ++dx) {
      if (dy == 0 && dx == 0) continue;
      const int yy = y + dy, xx = x + dx;
      if (yy < 0 || yy >= a.Dy || xx < 0 || xx >= a.Dx) continue;
      const float fn = F(dy, dx);
      // a neighbour at 0 above a negative F: masked (skipped by eq. 6) or a valid pixel that happens to hold 0?
      if (fn > fv && (fn != 0.f || a.W[(long long)yy * a.Dx + xx] != 0)) bigger = true;
    }
  return !bigger;
}

template <bool MASKED>
__device__ __forceinline__ bool peak_test_km(const FusedArgs& a, const float* __restrict__ X, int y, int x, float d, float s,
                                             float& fv, float& cc, float& se) {
  return a.k_max == 2 ? peak_test<2, MASKED>(a, X, y, x, d, s, fv, cc, se)
       : a.k_max == 1 ? peak_test<1, MASKED>(a, X, y, x, d, s, fv, cc, se)
                      : peak_test<0, MASKED>(a, X, y, x, d, s, fv, cc, se);
}

// grid (split, segments): the blocks of a segment share its entries.  A warp takes 32 entries at a time, spreads
// their surviving pixels over its lanes through shared memory (one pixel per lane and round) and appends the peaks
// with one atomic per round.
__global__ void __launch_bounds__(128)
k_peaks(const FusedArgs a) {
  __shared__ int s_pix[4][128];
  __shared__ float s_d[4][128], s_s[4][128];
  const int segi = blockIdx.y;
  const int p = segi / a.n_items;
  const int n = a.hit_cnt[segi];
  if ((int)(blockIdx.x * blockDim.x) >= n) return;
  const bool masked = *a.dirty == (a.fd ? a.fd->seq : a.dirty_seq);
  const long long N = (long long)a.Dy * a.Dx;
  const float* X = (p < a.B) ? (a.fd ? a.fd->cube : a.cube) + (long long)p * N : a.sum_plane;
  const HitRec* seg = a.hits + (long long)segi * a.seg_cap;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int i0 = blockIdx.x * blockDim.x; i0 < n; i0 += gridDim.x * blockDim.x) {
    const int i = i0 + threadIdx.x;
    int bits = 0, pix0 = 0;
    uint4 r1 = make_uint4(0u, 0u, 0u, 0u), r2 = r1;
    if (i < n) {
      const uint4* r = reinterpret_cast<const uint4*>(seg + i);
      const uint4 r0 = r[0];
      r1 = r[1]; r2 = r[2];
      pix0 = (int)r0.x; bits = (int)r0.y & 15;
    }
    // exclusive prefix of the pixel counts over the warp
    const int cnt = __popc(bits);
    int pre = cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const int v = __shfl_up_sync(0xffffffffu, pre, o); if (lane >= o) pre += v; }
    const int total = __shfl_sync(0xffffffffu, pre, 31);
    pre -= cnt;
    __syncwarp();
    {
      const uint32_t dk[4] = {r1.x, r1.y, r1.z, r1.w}, sk[4] = {r2.x, r2.y, r2.z, r2.w};
      int o = pre;
#pragma unroll
      for (int k = 0; k < 4; ++k)
        if ((bits >> k) & 1) { s_pix[warp][o] = pix0 + k; s_d[warp][o] = __uint_as_float(dk[k]); s_s[warp][o] = __uint_as_float(sk[k]); ++o; }
    }
    __syncwarp();
    for (int j0 = 0; j0 < total; j0 += 32) {
      const int j = j0 + lane;
      bool ok = false;
      int pix = 0;
      float d = 0.f, fv = 0.f, cc = 0.f, se = 1.f;
      if (j < total) {
        pix = s_pix[warp][j]; d = s_d[warp][j];
        const float sj = s_s[warp][j];
        const int y = pix / a.Dx, x = pix - y * a.Dx;
        ok = masked ? peak_test_km<true>(a, X, y, x, d, sj, fv, cc, se) : peak_test_km<false>(a, X, y, x, d, sj, fv, cc, se);
      }
      const unsigned m = __ballot_sync(0xffffffffu, ok);
      if (!m) continue;
      int base = 0;
      if (lane == 0) base = atomicAdd(a.ndets, __popc(m));
      base = __shfl_sync(0xffffffffu, base, 0);
      if (ok) {
        const int idx = base + __popc(m & ((1u << lane) - 1u));
        if (idx < a.max_det) {
          uint2* dst = reinterpret_cast<uint2*>(a.dets + idx);
          dst[0] = make_uint2((uint32_t)pix, (uint32_t)(p & 0xffff) | (1u << 16));        // int16 plane, int16 iter = 1
          dst[1] = make_uint2(__float_as_uint(fv), __float_as_uint(cc));
          dst[2] = make_uint2(__float_as_uint(se), __float_as_uint(d / sqrtf(se)));
        } else {
          atomicAdd(&a.counters[0], 1);
        }
      }
    }
    __syncwarp();
  }
}

}  // namespace

// ------------------------------------------------------------------------------------------------
// Work plan (host, once per context): column strips over the valid bounding box, row segments,
// the per-(iteration, warp) control words of every item, zero-padded normaliser planes.
struct LpfFusedPlan {
  bool ok = false;
  int CW = 0, NW = 0, threads = 0, n_items = 0, seg_cap = 0;
  size_t smem = 0;
  float nm_const = 1.f, ic_const = 1.f / 625.f;
  FusedItem* d_items = nullptr;
  uint32_t* d_flags = nullptr;
  float* d_nm_pad = nullptr;
  float* d_ic_pad = nullptr;
};

static size_t fused_smem_bytes(int NW) {
  const int CWP = NW * 128, XP = CWP + 8, PEV = CWP + 2 * KBG, PET = NW * 32 + 8;
  const size_t nfl = (size_t)XST * RB * XP + 4 * RB * PEV + 4 * RB * PET + 2 * XST + 2 + 2;
  return nfl * sizeof(float) + 16;
}

template <int NW>
static cudaError_t fused_launch_t(const FusedArgs& a, dim3 grid, size_t smem, cudaStream_t st, bool set_attr) {
  if (set_attr) return cudaFuncSetAttribute(k_sweep<NW>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  k_sweep<NW><<<grid, NW * 32 + 32, smem, st>>>(a);
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
  if (p.force_general) return LPF_OK;
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
    if (cw <= LPF_SWEEP_MAXW) { n_strips = (int)strips.size(); CW = cw; }
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
  // segments per strip: minimise waves x (rows per segment + warm-up cost) over the segment count.  With
  // n_lanes frames in flight the kernels of different lanes share the SMs, so each gets its share of them
  // (fewer, longer segments: less warm-up per output row).
  const int n_planes = c->n_planes;
  const int cta_per_sm = NW > 4 ? 1 : 2;      // k_sweep's launch bounds
  const int sm_share = std::max(1, cta_per_sm * c->n_sm / std::max(1, std::min(p.n_lanes, 4)));   // (more lanes in flight only deepen the queue;
                                                                                         // measured: 2 segments per plane beat 1 and 4)
  const double warm = 58.0;   // warm-up / drain rows of a segment
  int best_seg = 1; double best_cost = 1e30;
  const int max_rows_strip = (int)(rows_all / n_strips);
  for (int nseg = 1; nseg <= 64; ++nseg) {
    const double rows = (double)max_rows_strip / nseg;
    if (nseg > 1 && rows < 24) break;
    const long long ctas = (long long)nseg * n_strips * n_planes;
    const double waves = (double)((ctas + sm_share - 1) / sm_share);
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
    auto xmode = [&](int y, int w) -> unsigned { return ((cell(y, w) | cell(y + 1, w)) & CL_ANYW) ? FL_X : 0u; };
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
        f |= ld_bits(y0);
        if (b + 1 < it.nb) f |= ld_bits(y0 + RB) << 3;     // FL_*_LD -> FL_*_PF
        if (y0 + 1 - LAG_B >= it.ya - KBG) f |= FL_DO_B;
        if (y0 - LAG_C >= it.ya && y0 - LAG_C < it.yb) f |= FL_C0;
        if (y0 + 1 - LAG_C >= it.ya && y0 + 1 - LAG_C < it.yb) f |= FL_C1;
        flags.push_back(f);
      }
    ditems.push_back(it);
  }
  static_assert((FL_NM_LD << 3) == FL_NM_PF && (FL_ICR_LD << 3) == FL_ICR_PF && (FL_ICS_LD << 3) == FL_ICS_PF, "flag layout");

  LpfFusedPlan* pl = new LpfFusedPlan();
  pl->CW = CW; pl->NW = NW; pl->threads = NW * 32 + 32; pl->n_items = (int)ditems.size();
  pl->smem = fused_smem_bytes(NW);
  (void)max_nb;
  if ((long long)pl->n_items * c->n_planes > 65535) { delete pl; return LPF_OK; }   // grid.y of k_peaks
  {   // the hit list: HIT_BUDGET entries shared evenly by the (item, plane) segments
    const long long nseg = (long long)pl->n_items * c->n_planes;
    pl->seg_cap = (int)std::max<long long>(256, HIT_BUDGET / std::max<long long>(1, nseg));
  }
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

// rms-like scale of every plane for a cube whose QC statistics the caller kept to itself (lpf_detect_sources
// alone): sqrt(sum x^2 / n) over valid pixels x BIG_SIGMA.  One block per plane.
namespace {
__global__ void __launch_bounds__(1024)
k_big_thr(const float* __restrict__ cube, const float* __restrict__ sum_plane, const uint8_t* __restrict__ W, long long N, int B,
          float* __restrict__ big_thr) {
  __shared__ double s2[32], sn[32];
  const int p = blockIdx.x;
  const float* X = p < B ? cube + (long long)p * N : sum_plane;
  double a2 = 0, an = 0;
  for (long long i = threadIdx.x; i < N; i += blockDim.x)
    if (W[i]) { const float x = X[i]; a2 += (double)x * x; an += 1.0; }
  a2 = lpf_warp_sum(a2); an = lpf_warp_sum(an);
  if ((threadIdx.x & 31) == 0) { s2[threadIdx.x >> 5] = a2; sn[threadIdx.x >> 5] = an; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double t2 = 0, tn = 0;
    for (int w = 0; w < 32; ++w) { t2 += s2[w]; tn += sn[w]; }
    big_thr[p] = tn > 0 ? BIG_SIGMA * (float)sqrt(t2 / tn) : 0.f;
  }
}
}  // namespace

void lpf_fused_hit_sizes(const LpfFusedPlan* pl, int n_planes, long long* hit_bytes, long long* n_seg) {
  *n_seg = (long long)pl->n_items * n_planes;
  *hit_bytes = *n_seg * pl->seg_cap * (long long)sizeof(HitRec);
}

float lpf_fused_big_sigma(void) { return BIG_SIGMA; }

int lpf_launch_detect_fused(lpf_ctx* c, LpfFusedPlan* pl, LpfLane& L, const float* d_cube, const uint8_t* d_band_ok,
                            lpf_det* d_dets, int32_t* d_ndets, bool sum_done, cudaStream_t st) {
  const lpf_params& p = c->p;
  if (!sum_done) {     // the chained frame call has done all of this in its QC passes
    LPF_CUDA(cudaMemsetAsync(d_ndets, 0, sizeof(int32_t), st));
    int rc = lpf_launch_sum_plane(c, L, d_cube, d_band_ok, p.detect_sum_plane != 0, st);   // + the exact-zero check
    if (rc) return rc;
    LPF_KLAUNCH(c, KID_MISC, st, k_big_thr<<<c->n_planes, 1024, 0, st>>>(d_cube, L.sum_plane, c->W, c->N, p.B, L.big_thr));
  }
  FusedArgs a{};
  a.fd = c->cap_fd; a.cube = d_cube; a.sum_plane = L.sum_plane; a.band_ok = d_band_ok; a.W = c->W;
  a.nm_pad = pl->d_nm_pad; a.ic_pad = pl->d_ic_pad; a.items = pl->d_items; a.flags = pl->d_flags; a.dirty = L.dirty; a.dirty_seq = L.dirty_seq;
  a.big_thr = L.big_thr;
  a.B = p.B; a.Dy = p.Dy; a.Dx = p.Dx; a.CW = pl->CW; a.k_max = p.k_max; a.max_det = p.max_det; a.seg_cap = pl->seg_cap; a.n_items = pl->n_items;
  a.g0 = c->g_mf.g[3]; a.g1 = c->g_mf.g[2]; a.g2 = c->g_mf.g[1]; a.g3 = c->g_mf.g[0];
  a.kappa2 = p.kappa * p.kappa; a.eps_rel = p.eps_rel; a.nm_const = pl->nm_const; a.ic_const = pl->ic_const;
  a.hits = reinterpret_cast<HitRec*>(L.hits); a.hit_cnt = L.hit_cnt;
  a.dets = d_dets; a.ndets = d_ndets; a.counters = c->counters;
  const dim3 grid(pl->n_items, c->n_planes);
  LPF_KLAUNCH(c, KID_FUSED_DETECT, st, fused_dispatch(pl->NW, a, grid, pl->smem, st, false));
  {   // enough blocks per segment to cover the GPU a few times over; a block leaves at once when its share is empty
    const int nseg = pl->n_items * c->n_planes;
    const int split = std::max(1, std::min(64, (8 * c->n_sm + nseg - 1) / nseg));
    LPF_KLAUNCH(c, KID_PEAKS, st, k_peaks<<<dim3(split, nseg), 128, 0, st>>>(a));
  }
  return LPF_OK;
}
