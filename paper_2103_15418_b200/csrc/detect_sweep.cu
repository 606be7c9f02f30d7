// S4-S8 fused fast path: matched filter -> local centre -> local spread -> sigma clip -> local
// maxima -> compaction in ONE pass over each plane, for the headline parameter set
// (box background K = 12, Gaussian matched filter k_mf = 3, n_iter = 1).
// (eqs. 2-7; O3-O6 and "Sweep kernel".)
//
// Design (sm_100a).  A CTA owns a column strip (up to 1024 columns) and sweeps down a segment of rows.
// The three dependent stencil stages run in THREE GROUPS OF WARPS that hand rows to one another through
// shared-memory rings guarded by mbarriers (no block-wide barrier anywhere in the sweep), so the latency of
// one stage is covered by the work of the other two, and every thread owns 8 adjacent pixels (four packed
// f32x2 lanes of independent arithmetic):
//   A  rows y:        input rows arrive in a 4-stage shared ring by bulk asynchronous copies (TMA,
//                     cp.async.bulk + mbarrier) issued by a producer warp; horizontal 7-tap matched filter on the
//                     thread's 8 pixels (+3 either side), vertical 7-tap on a register window -> F(y-3) x norm_mf;
//                     25-row running sum V1 += F(y-3) - F(y-28); the V1 row goes to the V1 ring
//   B  rows rho=y-15: horizontal 25-box of the V1 row x 1/count -> C (eq. 3); d = F - C;
//                     running sum V2 += d^2 - d_old^2; the V2 row goes to the V2 ring, the F row (invalid
//                     pixels as -inf) to a 24-row shared ring for the local-maximum tests
//   C  rows sig=y-27: horizontal 25-box of the V2 row x 1/count -> S (eq. 4); eq. 5 for the warp's row is four
//                     packed operations, a max tree and one vote; the few hits apply the S_eff guard (R8), eq. 6
//                     on the shared F ring and append the eq. 7 record (one atomic per warp and row).
// The 32-row histories of F and d that the running sums and the lagged reads need are private to a pixel
// column, so they live in TENSOR MEMORY (tcgen05.st/ld 32x32b.x8): warp g of group A, B and C (warp ids g,
// g + 4, g + 8) share the 32 lanes g of the CTA's 512 columns: A writes the F ring, B reads it 12 rows
// later and writes the d ring, C reads that 12 rows later.  What a warp has to decide in a step (is there
// input, which normalisers are the interior constants, which stages run) is one 32-bit word of a per-item
// table built by the host plan.  F, C, d, S never leave the SM.
// The input is used unmasked when the cube holds exact zeros at every invalid pixel (checked per frame
// by the sum-plane kernel); otherwise each thread applies W itself (slow, rare).
// float32 running sums: V1 is safe for sources up to ~1e4 sigma; V2 = sum d^2 is
// re-summed exactly from the d ring whenever the roundings it has inherited (random walk: variance tracked
// per pixel as 2^-46/6 * sum of V2^2 over the rows since the last re-sum) could move S by more than 3e-5
// (1 sigma), i.e. when a bright source has just left the window, so it leaves nothing behind.
#include <algorithm>
#include <cstdio>
#include <cstdlib>

#include "lpf_internal.cuh"

extern __shared__ float4 g_sm4[];

namespace {

constexpr int KBG = 12;             // box half width
constexpr int WINB = 2 * KBG + 1;   // 25
constexpr int RB = 2;               // rows per step (the unit of hand-over between the warp groups)
constexpr int PX = 8;               // pixels per thread
constexpr int GW = 32 * PX;         // columns per warp: 256
constexpr int HALO = 2 * KBG + 3;   // rows of X above the first output row (27)
constexpr int LAG_B = 3 + KBG;      // rho = y - 15
constexpr int LAG_C = LAG_B + KBG;  // sig = y - 27
constexpr int DR = 32;              // depth (rows) of the tensor-memory rings of F and d (power of two)
constexpr int DF = 24;              // depth of the shared-memory ring of F rows (local maxima)
constexpr int XST = 4;              // input stages (steps in flight); = the number of register phases
constexpr int NV = 3;               // stages of the V1 and V2 rings
constexpr int TM_D = PX * DR;       // first tensor-memory column of the d ring (F ring starts at 0)
constexpr int PADR = 64;            // zero rows above and below the padded normaliser planes
constexpr int NTHREADS = 12 * 32;   // 4 A + 4 B + 4 C warps (lane 0 of the first A warp also issues the bulk copies)
constexpr float TRK_C = 2.56e-8f;  // V2 is re-summed when (sum of V2^2 over the rows since the last time) * TRK_C > V2^2

// per-(step, warp column) control word
constexpr unsigned FL_X = 1u;              // stage A has input: rows in the image, something valid near the warp
constexpr unsigned FL_NM_LD = 1u << 4;     // F rows of this step use the loaded norm_mf (else the constant)
constexpr unsigned FL_ICR_LD = 1u << 5;    // rho rows use the loaded 1/count
constexpr unsigned FL_ICS_LD = 1u << 6;    // sigma rows use the loaded 1/count
constexpr unsigned FL_NM_PF = 1u << 7;     // load the planes of the next step
constexpr unsigned FL_ICR_PF = 1u << 8;
constexpr unsigned FL_ICS_PF = 1u << 9;
constexpr unsigned FL_DO_B = 1u << 12;
constexpr unsigned FL_C0 = 1u << 13;       // sigma row j is an output row of this item
constexpr unsigned FL_C1 = 1u << 14;

struct FusedItem { int xs, ux0, ux1, ya, yb, y_start, nb, fl_off; };

struct FusedArgs {
  const float* cube; const float* sum_plane; const uint8_t* band_ok; const uint8_t* W;
  const float* nm_pad; const float* ic_pad;      // [(Dy + 2 PADR)][Dx], zero rows around the image
  const FusedItem* items; const uint32_t* flags;
  const int32_t* dirty; int dirty_seq;           // *dirty == dirty_seq: some invalid pixel of this cube is not an exact zero
  int B, Dy, Dx, CW, k_max, max_det;
  float g0, g1, g2, g3, kappa2, eps_rel, nm_const, ic_const;
  lpf_det* dets; int32_t* ndets; int32_t* counters;
};

__device__ __forceinline__ float4 zero4() { return make_float4(0.f, 0.f, 0.f, 0.f); }
// a global load the compiler may not sink to its use (the normaliser planes are fetched a step ahead)
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

// ---- tensor memory as a column-private scratch ring ------------------------------------------------
__device__ __forceinline__ void tm_st8(uint32_t taddr, const float2 (&v)[4]) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};\n"
               ::"r"(taddr), "f"(v[0].x), "f"(v[0].y), "f"(v[1].x), "f"(v[1].y), "f"(v[2].x), "f"(v[2].y), "f"(v[3].x), "f"(v[3].y));
}
__device__ __forceinline__ void tm_ld8(uint32_t taddr, float2 (&v)[4]) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];\n"
               : "=f"(v[0].x), "=f"(v[0].y), "=f"(v[1].x), "=f"(v[1].y), "=f"(v[2].x), "=f"(v[2].y), "=f"(v[3].x), "=f"(v[3].y)
               : "r"(taddr));
}
__device__ __forceinline__ void tm_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;\n"); }
__device__ __forceinline__ void tm_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;\n" ::: "memory"); }
__device__ __forceinline__ void tm_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory"); }
__device__ __forceinline__ void tm_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory"); }
// pins values loaded by tm_ld8 behind the tm_wait_ld that precedes this statement
__device__ __forceinline__ void tm_use(float2 (&v)[4]) {
  asm volatile("" : "+f"(v[0].x), "+f"(v[0].y), "+f"(v[1].x), "+f"(v[1].y), "+f"(v[2].x), "+f"(v[2].y), "+f"(v[3].x), "+f"(v[3].y));
}

// ---- bulk asynchronous copies (TMA without a tensor map) and mbarriers ---------------------------------
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
  // try_wait suspends the warp until the phase completes or the time hint runs out (no busy spinning)
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "LPF_WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1, %2;\n"
      "@p bra LPF_DONE_%=;\n"
      "bra LPF_WAIT_%=;\n"
      "LPF_DONE_%=:\n"
      "}\n" ::"r"(bar), "r"(parity), "r"(0x989680u) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n"
               ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}

// shared memory through the kernel's one dynamic array: float index -> value
__device__ __forceinline__ float4 lds4(int i) { return *reinterpret_cast<const float4*>(reinterpret_cast<const float*>(g_sm4) + i); }
__device__ __forceinline__ float lds1(int i) { return reinterpret_cast<const float*>(g_sm4)[i]; }
__device__ __forceinline__ void sts4(int i, float4 v) { *reinterpret_cast<float4*>(reinterpret_cast<float*>(g_sm4) + i) = v; }

// horizontal 25-box of a shared row for the thread's 8 pixels.  i0: float index of the value 12 columns to
// the left of the thread's first pixel; the 32 consecutive values v[0..31] = 16 aligned pairs Q_0..Q_15 cover all
// eight windows (pixel k: v[k..k+24]).  For the output pair p (pixels 2p, 2p+1) the 24 values v[2p+1..2p+24] are
// common: S_p = sum(Q_{p+1}..Q_{p+11}) + Q_p.y + Q_{p+12}.x, out = (S_p + Q_p.x, S_p + Q_{p+12}.y).  Sums only, all
// packed, no register shuffling (a swapped-halves operand is free).
__device__ __forceinline__ float2 swp(float2 a) { return make_float2(a.y, a.x); }
__device__ __forceinline__ void hbox25(int i0, float2 (&out)[4]) {
  float2 Q[16];
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const float4 q = lds4(i0 + 4 * i);
    Q[2 * i] = make_float2(q.x, q.y); Q[2 * i + 1] = make_float2(q.z, q.w);
  }
  const float2 K = add2(add2(add2(Q[4], Q[5]), add2(Q[6], Q[7])), add2(add2(Q[8], Q[9]), add2(Q[10], Q[11])));
  const float2 a = add2(Q[2], Q[3]), b = add2(Q[12], Q[13]);
  float2 W[4];
  W[0] = add2(K, add2(Q[1], a));
  W[1] = add2(K, add2(a, Q[12]));
  W[2] = add2(K, add2(Q[3], b));
  W[3] = add2(K, add2(b, Q[14]));
  const float2 e10 = make_float2(1.f, 0.f), e01 = make_float2(0.f, 1.f);
#pragma unroll
  for (int p = 0; p < 4; ++p) {
    const float2 T = add2(add2(W[p], swp(W[p])), add2(swp(Q[p]), Q[p + 12]));     // T.x = S_p
    out[p] = fma2(Q[p], e10, fma2(Q[p + 12], e01, splat(T.x)));
  }
}

// ---- shared-memory layout ---------------------------------------------------------------------------
template <int NG>
struct Lay {
  static constexpr int CWP = NG * GW;              // the CTA's full width
  static constexpr int XP = CWP + 8;               // staged input row: 4 columns of margin on both sides
  static constexpr int PV = CWP + 24;              // V1 / V2 row: 12 zero columns on both sides
  static constexpr int PF = CWP + 8;               // F row: 4 columns of -inf on both sides
  static constexpr int O_X = 0;
  static constexpr int O_V1 = O_X + XST * RB * XP;
  static constexpr int O_V2 = O_V1 + NV * RB * PV;
  static constexpr int O_FR = O_V2 + NV * RB * PV;
  static constexpr int O_FLG = O_FR + DF * PF;     // eq. 6 flags, one byte per thread and row, 32 rows
  static constexpr int O_BAR = O_FLG + 32 * NG * 32 / 4;     // mbarriers, 2 floats each
  static constexpr int B_FULL_X = 0, B_EMPTY_X = XST, B_FULL_V1 = 2 * XST, B_EMPTY_V1 = B_FULL_V1 + NV,
                       B_FULL_V2 = B_EMPTY_V1 + NV, B_EMPTY_V2 = B_FULL_V2 + NV, N_BAR = B_EMPTY_V2 + NV;
  static constexpr int O_END = O_BAR + 2 * N_BAR;
  __device__ static __forceinline__ uint32_t bar(int i) { return smem_u32(reinterpret_cast<const float*>(g_sm4) + O_BAR + 2 * i); }
};

// what every role needs
struct Ctx {
  const FusedArgs* a;      // kernel arguments (shared-memory copy)
  int xs, plane, lane, g, t;     // strip origin, plane, lane, warp column, thread index within the row (g * 32 + lane)
  int nb;
  const uint32_t* flp;     // this warp column's control words, [nb] with stride NG
  int sx;                  // row stride of the plane pointers (0 for lanes outside the strip)
  uint32_t tm;             // tensor-memory address of the thread's ring column 0
};

template <int NG>
__device__ __forceinline__ unsigned ctl(const Ctx& c, int b) {
  unsigned v = 0u;
  if (b < c.nb) asm volatile("ld.global.nc.u32 %0, [%1];\n" : "=r"(v) : "l"(c.flp + b * NG));
  return v;
}

// ring stage counter with its phase parity
struct Stage {
  int s = 0; uint32_t par = 0;
  __device__ __forceinline__ void next(int n) { if (++s == n) { s = 0; par ^= 1u; } }
};

// ---- group A: matched filter and the running sum of F --------------------------------------------------
// the slow input path: a cube with something other than an exact zero at an invalid pixel; x0: image column of v[0]
struct Row16 { float v[16]; };
__device__ __noinline__ Row16 mask_row16(const FusedArgs* ap, int y, int x0, Row16 r) {
  const FusedArgs& a = *ap;
#pragma unroll
  for (int k = 0; k < 16; ++k) {
    const int x = x0 + k;
    const bool ok = y >= 0 && y < a.Dy && x >= 0 && x < a.Dx && a.W[(long long)y * a.Dx + x] != 0;
    if (!ok) r.v[k] = 0.f;
  }
  return r;
}

template <int NG>
struct RoleA {
  using L = Lay<NG>;
  const Ctx c;
  const FusedArgs& a;
  bool dirty;
  int y0;                  // first input row of the current step
  const float* nmp;        // padded norm_mf at the next step's first F row
  float2 hw[8][4];         // horizontally filtered rows (rotating; static indices per phase)
  float2 V1[4];            // vertical running sum of F
  float4 nm[RB][2];        // normalisers of the coming rows
  Stage sv;                // V1 ring stage
  // producer (lane 0 of the first A warp): the input rows of step bb go into stage bb mod XST
  bool producer;
  const float* xrow0;      // X at (y_start, first copied column)
  uint32_t x_dst0;         // shared address of that column in stage 0, row 0
  uint32_t row_bytes;
  int ys;

  // the two input rows of step bb into stage bb mod XST (a plain arrival when they lie outside the image)
  __device__ __forceinline__ void issue_rows(int bb) {
    const int st = bb & (XST - 1);
    const int y = ys + RB * bb;
    if (bb >= XST) mbar_wait(L::bar(L::B_EMPTY_X + st), (uint32_t)((bb >> 2) - 1) & 1u);   // every A warp has read its previous content
    const uint32_t bar = L::bar(L::B_FULL_X + st);
    if (y >= 0 && y + RB <= a.Dy) {
      mbar_expect_tx(bar, RB * row_bytes);
      const float* src = xrow0 + (long long)RB * bb * a.Dx;
      const uint32_t dst = x_dst0 + (uint32_t)(st * RB * L::XP * 4);
#pragma unroll
      for (int j = 0; j < RB; ++j) bulk_g2s(dst + (uint32_t)(j * L::XP * 4), src + (long long)j * a.Dx, row_bytes, bar);
    } else {
      mbar_arrive(bar);
    }
  }

  __device__ __forceinline__ RoleA(const Ctx& c_, const FusedArgs& a_) : c(c_), a(a_) {}

  __device__ __forceinline__ void load_nm(unsigned on) {
    if (on) {
#pragma unroll
      for (int j = 0; j < RB; ++j) { nm[j][0] = ldg4_pinned(nmp + j * c.sx); nm[j][1] = ldg4_pinned(nmp + j * c.sx + 4); }
    }
    nmp += RB * c.sx;
  }

  template <int PH>
  __device__ __forceinline__ void step(int s, unsigned fl) {
    const float2 g0 = splat(a.g0), g1 = splat(a.g1), g2 = splat(a.g2), g3 = splat(a.g3);
    const float2 c30 = make_float2(a.g3, 0.f), c13 = make_float2(a.g1, a.g3), c31 = make_float2(a.g3, a.g1), c03 = make_float2(0.f, a.g3);
    const uint32_t w0 = (uint32_t)(RB * s) & (DR - 1);
    const uint32_t t_new0 = c.tm + PX * w0, t_new1 = t_new0 + PX;
    const uint32_t t_old0 = c.tm + PX * ((w0 + 7) & (DR - 1)), t_old1 = c.tm + PX * ((w0 + 8) & (DR - 1));
    float2 fold[RB][4];
    tm_ld8(t_old0, fold[0]); tm_ld8(t_old1, fold[1]);          // F(fr - 25)

    if (producer && s + XST - 1 < c.nb) issue_rows(s + XST - 1);   // its stage was read in step s - 1
    // ---- staged input rows -> horizontal matched filter -> hw ------------------------------------------
    mbar_wait(L::bar(L::B_FULL_X + PH), (uint32_t)(s >> 2) & 1u);
    if (fl & FL_X) {
#pragma unroll
      for (int j = 0; j < RB; ++j) {
        const int xr = L::O_X + (PH * RB + j) * L::XP + PX * c.t;
        const float4 q0 = lds4(xr), q1 = lds4(xr + 4), q2 = lds4(xr + 8), q3 = lds4(xr + 12);
        float v[16] = {q0.x, q0.y, q0.z, q0.w, q1.x, q1.y, q1.z, q1.w, q2.x, q2.y, q2.z, q2.w, q3.x, q3.y, q3.z, q3.w};
        if (dirty) {
          Row16 r;
#pragma unroll
          for (int k = 0; k < 16; ++k) r.v[k] = v[k];
          r = mask_row16(c.a, y0 + j, c.xs + PX * c.t - 4, r);
#pragma unroll
          for (int k = 0; k < 16; ++k) v[k] = r.v[k];
        }
        // pixel k of the thread is v[k + 4]: aligned input pairs P_m = (v[2m], v[2m+1]); output pair p <- P_{p..p+4}.
        // With sw() the swapped pair: O_p = g2 (P_{p+1} + P_{p+3}) + g0 P_{p+2}
        //   + (g3,0) sw(P_p) + (g1,g3) sw(P_{p+1}) + (g1,g1) sw(P_{p+2}) + (g3,g1) sw(P_{p+3}) + (0,g3) sw(P_{p+4}):
        // every operand is an aligned register pair (swapping halves is free), no register moves.
        float2 P[8];
#pragma unroll
        for (int m = 0; m < 8; ++m) P[m] = make_float2(v[2 * m], v[2 * m + 1]);
#pragma unroll
        for (int p = 0; p < 4; ++p) {
          float2 o = mul2(c30, swp(P[p]));
          o = fma2(c13, swp(P[p + 1]), o);
          o = fma2(g1, swp(P[p + 2]), o);
          o = fma2(c31, swp(P[p + 3]), o);
          o = fma2(c03, swp(P[p + 4]), o);
          o = fma2(g2, add2(P[p + 1], P[p + 3]), o);
          hw[(2 * PH + 6 + j) & 7][p] = fma2(g0, P[p + 2], o);
        }
      }
    } else {
#pragma unroll
      for (int j = 0; j < RB; ++j)
#pragma unroll
        for (int p = 0; p < 4; ++p) hw[(2 * PH + 6 + j) & 7][p] = splat(0.f);
    }
    __syncwarp();
    if (c.lane == 0) mbar_arrive(L::bar(L::B_EMPTY_X + PH));    // the stage may be refilled

    // ---- vertical matched filter -> F(fr), running sum V1, hand-over ---------------------------------
    float2 f[RB][4];
#pragma unroll
    for (int j = 0; j < RB; ++j)
#pragma unroll
      for (int p = 0; p < 4; ++p) {
        const float2 h0 = hw[(2 * PH + j + 0) & 7][p], h1 = hw[(2 * PH + j + 1) & 7][p], h2 = hw[(2 * PH + j + 2) & 7][p],
                     h3 = hw[(2 * PH + j + 3) & 7][p], h4 = hw[(2 * PH + j + 4) & 7][p], h5 = hw[(2 * PH + j + 5) & 7][p],
                     h6 = hw[(2 * PH + j + 6) & 7][p];
        f[j][p] = fma2(g0, h3, fma2(g1, add2(h2, h4), fma2(g2, add2(h1, h5), mul2(g3, add2(h0, h6)))));
      }
    if (fl & FL_NM_LD) {
#pragma unroll
      for (int j = 0; j < RB; ++j) {
        f[j][0] = mul2(f[j][0], make_float2(nm[j][0].x, nm[j][0].y)); f[j][1] = mul2(f[j][1], make_float2(nm[j][0].z, nm[j][0].w));
        f[j][2] = mul2(f[j][2], make_float2(nm[j][1].x, nm[j][1].y)); f[j][3] = mul2(f[j][3], make_float2(nm[j][1].z, nm[j][1].w));
      }
    } else {
      const float2 k = splat(a.nm_const);
#pragma unroll
      for (int j = 0; j < RB; ++j)
#pragma unroll
        for (int p = 0; p < 4; ++p) f[j][p] = mul2(f[j][p], k);
    }
    load_nm(fl & FL_NM_PF);                          // the next step's norm_mf rows
    tm_wait_ld();
    tm_use(fold[0]); tm_use(fold[1]);
    if (s >= NV) mbar_wait(L::bar(L::B_EMPTY_V1 + sv.s), sv.par ^ 1u);      // group B is done with this stage
#pragma unroll
    for (int j = 0; j < RB; ++j) {
#pragma unroll
      for (int p = 0; p < 4; ++p) V1[p] = add2(V1[p], sub2(f[j][p], fold[j][p]));
      tm_st8(j ? t_new1 : t_new0, f[j]);
      const int o = L::O_V1 + (sv.s * RB + j) * L::PV + KBG + PX * c.t;
      sts4(o, make_float4(V1[0].x, V1[0].y, V1[1].x, V1[1].y));
      sts4(o + 4, make_float4(V1[2].x, V1[2].y, V1[3].x, V1[3].y));
    }
    tm_wait_st();
    tm_fence_before();
    __syncwarp();
    if (c.lane == 0) mbar_arrive(L::bar(L::B_FULL_V1 + sv.s));
    sv.next(NV);
    y0 += RB;
  }

  __device__ __forceinline__ void run() {
    {
      const unsigned f0 = ctl<NG>(c, 0);
      load_nm(f0 & FL_NM_LD);
    }
    if (producer)
      for (int bb = 0; bb < XST - 1 && bb < c.nb; ++bb) issue_rows(bb);
    int b = 0;
    unsigned f0 = ctl<NG>(c, 0), f1 = ctl<NG>(c, 1), f2 = ctl<NG>(c, 2), f3;
    while (true) {
      f3 = ctl<NG>(c, b + 3);
      step<0>(b, f0); if (++b >= c.nb) break;
      f0 = ctl<NG>(c, b + 3);
      step<1>(b, f1); if (++b >= c.nb) break;
      f1 = ctl<NG>(c, b + 3);
      step<2>(b, f2); if (++b >= c.nb) break;
      f2 = ctl<NG>(c, b + 3);
      step<3>(b, f3); if (++b >= c.nb) break;
    }
  }
};

// ---- group B: local centre, residual, running sum of the squared residual ----------------------------------
// exact re-sum of V2 = sum over the 25 rows rho-24 .. rho of d^2 from the tensor-memory ring; slot: ring slot of rho
struct Acc4 { float2 v[4]; };
__device__ __noinline__ Acc4 resum_v2(uint32_t tm_d, uint32_t slot) {
  float2 acc[4] = {splat(0.f), splat(0.f), splat(0.f), splat(0.f)};
  for (int i0 = WINB - 1; i0 >= 0; i0 -= 5) {       // oldest first, five rows in flight
    float2 d[5][4];
#pragma unroll
    for (int k = 0; k < 5; ++k) tm_ld8(tm_d + PX * ((slot + DR - (i0 - k)) & (DR - 1)), d[k]);
    tm_wait_ld();
#pragma unroll
    for (int k = 0; k < 5; ++k) {
      tm_use(d[k]);
#pragma unroll
      for (int p = 0; p < 4; ++p) acc[p] = fma2(d[k][p], d[k][p], acc[p]);
    }
  }
  Acc4 r;
#pragma unroll
  for (int p = 0; p < 4; ++p) r.v[p] = acc[p];
  return r;
}

template <int NG>
struct RoleB {
  using L = Lay<NG>;
  const Ctx c;
  const FusedArgs& a;
  const float* icp;        // padded 1/count at the next step's first rho row
  float2 V2[4], E[4];      // running sum of d^2; sum of V2^2 over the rows since the last exact re-sum
  float2 Fw[6][4];         // the F rows (invalid pixels -inf) of this step and the two before (rotating, 3 phases)
  float4 ic[RB][2];
  Stage sv;                // stage of both rings (V1 consumed, V2 produced: same step index)
  int fr;                  // F-ring slot of this step's first rho row
  int fq;                  // flag-ring row of rho0 - 2 (the first row whose eq. 6 flags this step settles)

  __device__ __forceinline__ RoleB(const Ctx& c_, const FusedArgs& a_) : c(c_), a(a_) {}

  __device__ __forceinline__ void load_ic(unsigned on) {
    if (on) {
#pragma unroll
      for (int j = 0; j < RB; ++j) { ic[j][0] = ldg4_pinned(icp + j * c.sx); ic[j][1] = ldg4_pinned(icp + j * c.sx + 4); }
    }
    icp += RB * c.sx;
  }

  template <int PH3>
  __device__ __forceinline__ void step(int s, unsigned fl) {
    constexpr int WN = 2 * PH3, WP = 2 * ((PH3 + 2) % 3), WPP = 2 * ((PH3 + 1) % 3);   // window rows: new, previous step, the one before
    const uint32_t w0 = (uint32_t)(RB * s) & (DR - 1);
    const uint32_t t_lag0 = c.tm + PX * ((w0 + 20) & (DR - 1)), t_lag1 = t_lag0 + PX;       // F(rho): w0 + 20 is even
    const uint32_t t_new0 = c.tm + TM_D + PX * w0, t_new1 = t_new0 + PX;
    const uint32_t t_old0 = c.tm + TM_D + PX * ((w0 + 7) & (DR - 1)), t_old1 = c.tm + TM_D + PX * ((w0 + 8) & (DR - 1));
    mbar_wait(L::bar(L::B_FULL_V1 + sv.s), sv.par);
    tm_fence_after();
    float2 F[RB][4], dold[RB][4], bx[RB][4];
    tm_ld8(t_lag0, F[0]); tm_ld8(t_lag1, F[1]);
    tm_ld8(t_old0, dold[0]); tm_ld8(t_old1, dold[1]);
#pragma unroll
    for (int j = 0; j < RB; ++j) hbox25(L::O_V1 + (sv.s * RB + j) * L::PV + PX * c.t, bx[j]);
    __syncwarp();
    if (c.lane == 0) mbar_arrive(L::bar(L::B_EMPTY_V1 + sv.s));
    tm_wait_ld();
    tm_use(F[0]); tm_use(F[1]); tm_use(dold[0]); tm_use(dold[1]);
    if (s >= NV) mbar_wait(L::bar(L::B_EMPTY_V2 + sv.s), sv.par ^ 1u);      // group C is done with this stage
    if (fl & FL_DO_B) {
#pragma unroll
      for (int j = 0; j < RB; ++j) {
        float2 dd[4], fm[4];
        if (fl & FL_ICR_LD) {
          const float2 i0 = make_float2(ic[j][0].x, ic[j][0].y), i1 = make_float2(ic[j][0].z, ic[j][0].w),
                       i2 = make_float2(ic[j][1].x, ic[j][1].y), i3 = make_float2(ic[j][1].z, ic[j][1].w);
          dd[0] = fma2(neg2(bx[j][0]), i0, F[j][0]); dd[1] = fma2(neg2(bx[j][1]), i1, F[j][1]);     // d = F - box * (1/count)
          dd[2] = fma2(neg2(bx[j][2]), i2, F[j][2]); dd[3] = fma2(neg2(bx[j][3]), i3, F[j][3]);
          const float ninf = __int_as_float(0xff800000);
          // 1/count is 0 exactly at invalid pixels (and outside the image): they never win a local-maximum test
          fm[0] = make_float2(i0.x != 0.f ? F[j][0].x : ninf, i0.y != 0.f ? F[j][0].y : ninf);
          fm[1] = make_float2(i1.x != 0.f ? F[j][1].x : ninf, i1.y != 0.f ? F[j][1].y : ninf);
          fm[2] = make_float2(i2.x != 0.f ? F[j][2].x : ninf, i2.y != 0.f ? F[j][2].y : ninf);
          fm[3] = make_float2(i3.x != 0.f ? F[j][3].x : ninf, i3.y != 0.f ? F[j][3].y : ninf);
        } else {
          const float2 k = splat(a.ic_const);
#pragma unroll
          for (int p = 0; p < 4; ++p) { dd[p] = fma2(neg2(bx[j][p]), k, F[j][p]); fm[p] = F[j][p]; }
        }
#pragma unroll
        for (int p = 0; p < 4; ++p) {
          V2[p] = fma2(neg2(dold[j][p]), dold[j][p], fma2(dd[p], dd[p], V2[p]));
          E[p] = fma2(V2[p], V2[p], E[p]);
        }
        tm_st8(j ? t_new1 : t_new0, dd);
        const int o = L::O_V2 + (sv.s * RB + j) * L::PV + KBG + PX * c.t;
        sts4(o, make_float4(V2[0].x, V2[0].y, V2[1].x, V2[1].y));
        sts4(o + 4, make_float4(V2[2].x, V2[2].y, V2[3].x, V2[3].y));
#pragma unroll
        for (int p = 0; p < 4; ++p) Fw[WN + j][p] = fm[p];
      }
      {   // eq. 6, vertical half, for the two rows of the previous step (centres q = rho0 - 2, rho0 - 1: their windows are
          // complete now): cm = the column maximum over rows q-k_max .. q+k_max goes to the shared ring (group C compares
          // it across columns), and one bit per pixel says whether F(q, x) is that maximum (then cm IS F(q, x))
        const int km = a.k_max;
        uint8_t* flg = reinterpret_cast<uint8_t*>(reinterpret_cast<float*>(g_sm4) + L::O_FLG);
#pragma unroll
        for (int j = 0; j < RB; ++j) {
          float2 cm[4];
          unsigned q = 0u;
#pragma unroll
          for (int p = 0; p < 4; ++p) {
            // rows around the centre WP + j: one up / down, two up / down (window slots of the three steps)
            const float2 ce = Fw[WP + j][p];
            const float2 u1 = j ? Fw[WP][p] : Fw[WPP + 1][p], d1 = j ? Fw[WN][p] : Fw[WP + 1][p];
            const float2 u2 = j ? Fw[WPP + 1][p] : Fw[WPP][p], d2 = j ? Fw[WN + 1][p] : Fw[WN][p];
            float2 x = ce;
            if (km >= 1) x = make_float2(fmaxf(x.x, fmaxf(u1.x, d1.x)), fmaxf(x.y, fmaxf(u1.y, d1.y)));
            if (km >= 2) x = make_float2(fmaxf(x.x, fmaxf(u2.x, d2.x)), fmaxf(x.y, fmaxf(u2.y, d2.y)));
            cm[p] = x;
            q |= (ce.x >= x.x ? 1u : 0u) << (2 * p);
            q |= (ce.y >= x.y ? 1u : 0u) << (2 * p + 1);
          }
          int sl = fr + j - 2; sl = sl < 0 ? sl + DF : sl;
          const int of = L::O_FR + sl * L::PF + 4 + PX * c.t;
          sts4(of, make_float4(cm[0].x, cm[0].y, cm[1].x, cm[1].y));
          sts4(of + 4, make_float4(cm[2].x, cm[2].y, cm[3].x, cm[3].y));
          flg[((fq + j) & 31) * (NG * 32) + c.t] = (uint8_t)q;
        }
      }
      // the roundings V2 has inherited: variance 2^-46/6 * sum of V2^2 over the rows since the last exact re-sum
      float2 tq[4];
#pragma unroll
      for (int p = 0; p < 4; ++p) tq[p] = fma2(E[p], splat(TRK_C), neg2(mul2(V2[p], V2[p])));
      const float worst = fmaxf(fmaxf(fmaxf(tq[0].x, tq[0].y), fmaxf(tq[1].x, tq[1].y)), fmaxf(fmaxf(tq[2].x, tq[2].y), fmaxf(tq[3].x, tq[3].y)));
      if (__any_sync(0xffffffffu, worst > 0.f)) {
        tm_wait_st();
        const Acc4 r = resum_v2(c.tm + TM_D, (w0 + 1) & (DR - 1));
#pragma unroll
        for (int p = 0; p < 4; ++p) V2[p] = r.v[p];
        // the rows already handed over keep the incremental value (inside the bound by construction); the next rows start clean
#pragma unroll
        for (int p = 0; p < 4; ++p) E[p] = splat(0.f);
      }
    }
    load_ic(fl & FL_ICR_PF);
    tm_wait_st();
    tm_fence_before();
    __syncwarp();
    if (c.lane == 0) mbar_arrive(L::bar(L::B_FULL_V2 + sv.s));
    sv.next(NV);
    fr += RB; fr = fr >= DF ? fr - DF : fr;
    fq += RB;
  }

  __device__ __forceinline__ void run() {
    {
      const unsigned f0 = ctl<NG>(c, 0);
      load_ic(f0 & FL_ICR_LD);
    }
    unsigned f0 = ctl<NG>(c, 0), f1 = ctl<NG>(c, 1), f2 = ctl<NG>(c, 2);
    int b = 0;
    while (true) {     // the word of step b + 3 takes the place of the one just used
      step<0>(b, f0); f0 = ctl<NG>(c, b + 3); if (++b >= c.nb) break;
      step<1>(b, f1); f1 = ctl<NG>(c, b + 3); if (++b >= c.nb) break;
      step<2>(b, f2); f2 = ctl<NG>(c, b + 3); if (++b >= c.nb) break;
    }
  }
};

// ---- group C: local spread, eq. 5, and for the hits eq. 6 / eq. 7 ------------------------------------------
// The pixels flagged in `bits` (one byte per lane) passed the unguarded eq. 5 and the vertical half of eq. 6 (group B's
// flag: F is the maximum of its column over the window's rows, so the ring value cm at that pixel IS F).  What is left:
// the horizontal half, cm(x) >= cm(x + dx) for |dx| <= k_max on the shared ring row (invalid pixels and the margins
// hold -inf), the S_eff guard (R8) and eq. 5 in its rounded form.  The records of the warp's row go to the global list
// with one atomic.  row0: float index of the lane's first pixel in the ring row of sigma; cl: its strip column.
__device__ __noinline__ void c_hits(const FusedArgs* ap, int row0, int cl, int sg, int xs, int plane, int lane, unsigned bits,
                                    float4 d0, float4 d1, float4 s0, float4 s1) {
  const FusedArgs& a = *ap;
  const int km = a.k_max;
  float cm[12];                                      // columns -2 .. 9 relative to the lane's first pixel
  {
    const float4 q0 = lds4(row0), q1 = lds4(row0 + 4);
    const float2 ql = *reinterpret_cast<const float2*>(reinterpret_cast<const float*>(g_sm4) + row0 - 2);
    const float2 qr = *reinterpret_cast<const float2*>(reinterpret_cast<const float*>(g_sm4) + row0 + 8);
    cm[0] = ql.x; cm[1] = ql.y; cm[2] = q0.x; cm[3] = q0.y; cm[4] = q0.z; cm[5] = q0.w;
    cm[6] = q1.x; cm[7] = q1.y; cm[8] = q1.z; cm[9] = q1.w; cm[10] = qr.x; cm[11] = qr.y;
  }
  const float d[8] = {d0.x, d0.y, d0.z, d0.w, d1.x, d1.y, d1.z, d1.w};
  const float sv[8] = {s0.x, s0.y, s0.z, s0.w, s1.x, s1.y, s1.z, s1.w};
  unsigned ok = 0u;
  float se[8];
#pragma unroll
  for (int k = 0; k < 8; ++k) {
    const float f = cm[k + 2];
    float nb = __int_as_float(0xff800000);
    if (km >= 1) nb = fmaxf(cm[k + 1], cm[k + 3]);
    if (km >= 2) nb = fmaxf(nb, fmaxf(cm[k], cm[k + 4]));
    const float cc = f - d[k];
    const float gd = a.eps_rel * fabsf(cc);
    const float sef = fmaxf(sv[k], gd * gd);
    se[k] = sef;
    if (((bits >> k) & 1u) && !(nb > f) && d[k] > 0.f && d[k] * d[k] > a.kappa2 * sef) ok |= 1u << k;
  }
  // append: exclusive prefix of the lanes' counts, one atomic for the warp
  const int n = __popc(ok);
  int incl = n;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const int v = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += v; }
  const int total = __shfl_sync(0xffffffffu, incl, 31);
  if (total == 0) return;
  int base = 0;
  if (lane == 0) base = atomicAdd(a.ndets, total);
  base = __shfl_sync(0xffffffffu, base, 0);
  int idx = base + incl - n;
#pragma unroll
  for (int k = 0; k < 8; ++k) {
    if (!((ok >> k) & 1u)) continue;
    if (idx < a.max_det) {
      uint2* dst = reinterpret_cast<uint2*>(a.dets + idx);
      dst[0] = make_uint2((uint32_t)(sg * a.Dx + xs + cl + k), (uint32_t)(plane & 0xffff) | (1u << 16));   // int16 plane, int16 iter = 1
      dst[1] = make_uint2(__float_as_uint(cm[k + 2]), __float_as_uint(cm[k + 2] - d[k]));
      dst[2] = make_uint2(__float_as_uint(se[k]), __float_as_uint(d[k] / sqrtf(se[k])));
    } else {
      atomicAdd(&a.counters[0], 1);
    }
    ++idx;
  }
}

template <int NG>
struct RoleC {
  using L = Lay<NG>;
  const Ctx c;
  const FusedArgs& a;
  const float* icp;        // padded 1/count at the next step's first sigma row
  float4 ic[RB][2];
  Stage sv;
  int fr;                  // F-ring slot of this step's first sigma row
  int y0;                  // first input row of the current step (sigma = y0 + j - LAG_C)
  unsigned umask;          // the thread's pixels that this item outputs

  __device__ __forceinline__ RoleC(const Ctx& c_, const FusedArgs& a_) : c(c_), a(a_) {}

  __device__ __forceinline__ void load_ic(unsigned on) {
    if (on) {
#pragma unroll
      for (int j = 0; j < RB; ++j) { ic[j][0] = ldg4_pinned(icp + j * c.sx); ic[j][1] = ldg4_pinned(icp + j * c.sx + 4); }
    }
    icp += RB * c.sx;
  }

  __device__ __forceinline__ void step(int s, unsigned fl) {
    const uint32_t w0 = (uint32_t)(RB * s) & (DR - 1);
    const uint32_t t_lag0 = c.tm + TM_D + PX * ((w0 + 20) & (DR - 1)), t_lag1 = t_lag0 + PX;       // d(sigma)
    mbar_wait(L::bar(L::B_FULL_V2 + sv.s), sv.par);
    tm_fence_after();
    if (fl & (FL_C0 | FL_C1)) {
      float2 dl[RB][4], bx[RB][4];
      tm_ld8(t_lag0, dl[0]); tm_ld8(t_lag1, dl[1]);
#pragma unroll
      for (int j = 0; j < RB; ++j) hbox25(L::O_V2 + (sv.s * RB + j) * L::PV + PX * c.t, bx[j]);
      __syncwarp();
      if (c.lane == 0) mbar_arrive(L::bar(L::B_EMPTY_V2 + sv.s));
      tm_wait_ld();
      tm_use(dl[0]); tm_use(dl[1]);
#pragma unroll
      for (int j = 0; j < RB; ++j) {
        if (!(fl & (FL_C0 << j))) continue;          // uniform
        float2 S[4], m[4];
        if (fl & FL_ICS_LD) {
          S[0] = mul2(bx[j][0], make_float2(ic[j][0].x, ic[j][0].y)); S[1] = mul2(bx[j][1], make_float2(ic[j][0].z, ic[j][0].w));
          S[2] = mul2(bx[j][2], make_float2(ic[j][1].x, ic[j][1].y)); S[3] = mul2(bx[j][3], make_float2(ic[j][1].z, ic[j][1].w));
        } else {
          const float2 k = splat(a.ic_const);
#pragma unroll
          for (int p = 0; p < 4; ++p) S[p] = mul2(bx[j][p], k);
        }
        // d^2 - kappa^2 S > 0 somewhere in the warp's row?  (the sign of the fused difference is exact)
        const float2 nk2 = splat(-a.kappa2);
#pragma unroll
        for (int p = 0; p < 4; ++p) m[p] = fma2(dl[j][p], dl[j][p], mul2(S[p], nk2));
        const float mm = fmaxf(fmaxf(fmaxf(m[0].x, m[0].y), fmaxf(m[1].x, m[1].y)), fmaxf(fmaxf(m[2].x, m[2].y), fmaxf(m[3].x, m[3].y)));
        if (__any_sync(0xffffffffu, mm > 0.f)) {
          const float dv[8] = {dl[j][0].x, dl[j][0].y, dl[j][1].x, dl[j][1].y, dl[j][2].x, dl[j][2].y, dl[j][3].x, dl[j][3].y};
          const float mv[8] = {m[0].x, m[0].y, m[1].x, m[1].y, m[2].x, m[2].y, m[3].x, m[3].y};
          unsigned bits = 0u;
#pragma unroll
          for (int k = 0; k < 8; ++k)
            if (dv[k] > 0.f && mv[k] > 0.f) bits |= 1u << k;
          {   // group B's flags of row sigma: the vertical half of eq. 6 (written 10 rows ago)
            const uint8_t* flg = reinterpret_cast<const uint8_t*>(reinterpret_cast<const float*>(g_sm4) + L::O_FLG);
            bits &= umask & (unsigned)flg[((RB * s + j + 20) & 31) * (NG * 32) + c.t];
          }
          if (__any_sync(0xffffffffu, bits != 0u)) {
            int sl = fr + j; sl = sl >= DF ? sl - DF : sl;
            c_hits(c.a, L::O_FR + 4 + sl * L::PF + PX * c.t, PX * c.t, y0 + j - LAG_C, c.xs, c.plane, c.lane, bits,
                          make_float4(dl[j][0].x, dl[j][0].y, dl[j][1].x, dl[j][1].y), make_float4(dl[j][2].x, dl[j][2].y, dl[j][3].x, dl[j][3].y),
                          make_float4(S[0].x, S[0].y, S[1].x, S[1].y), make_float4(S[2].x, S[2].y, S[3].x, S[3].y));
          }
        }
      }
    } else {
      __syncwarp();
      if (c.lane == 0) mbar_arrive(L::bar(L::B_EMPTY_V2 + sv.s));
    }
    load_ic(fl & FL_ICS_PF);
    sv.next(NV);
    fr += RB; fr = fr >= DF ? fr - DF : fr;
    y0 += RB;
  }

  __device__ __forceinline__ void run() {
    {
      const unsigned f0 = ctl<NG>(c, 0);
      load_ic(f0 & FL_ICS_LD);
    }
    unsigned f0 = ctl<NG>(c, 0), f1 = ctl<NG>(c, 1), f2 = ctl<NG>(c, 2);
    for (int b = 0; b < c.nb; ++b) {
      const unsigned f3 = ctl<NG>(c, b + 3);
      step(b, f0);
      f0 = f1; f1 = f2; f2 = f3;
    }
  }
};

template <int NG>
__global__ void __launch_bounds__(NTHREADS, 1)
k_sweep_box(const FusedArgs a) {
  __shared__ uint32_t s_tmem;
  __shared__ FusedArgs s_args;
  using L = Lay<NG>;
  const int p = blockIdx.y;
  if (!a.band_ok[a.B]) return;
  if (p < a.B && !a.band_ok[p]) return;

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const FusedItem it = a.items[blockIdx.x];
  if (tid == 0) s_args = a;
  for (int i = tid; i < (L::O_END + 3) / 4; i += NTHREADS) g_sm4[i] = zero4();
  __syncthreads();
  {   // the F ring starts as -inf everywhere (its margins stay so: columns outside the strip never win)
    const float ninf = __int_as_float(0xff800000);
    const float4 n4 = make_float4(ninf, ninf, ninf, ninf);
    for (int i = tid; i < DF * L::PF / 4; i += NTHREADS) g_sm4[L::O_FR / 4 + i] = n4;
  }
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;\n"
                 ::"l"((uint64_t)__cvta_generic_to_shared(&s_tmem)), "n"(512));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n");
  }
  if (tid == 0) {
#pragma unroll
    for (int i = 0; i < XST; ++i) { mbar_init(L::bar(L::B_FULL_X + i), 1); mbar_init(L::bar(L::B_EMPTY_X + i), NG); }
#pragma unroll
    for (int i = 0; i < NV; ++i) {
      mbar_init(L::bar(L::B_FULL_V1 + i), NG); mbar_init(L::bar(L::B_EMPTY_V1 + i), NG);
      mbar_init(L::bar(L::B_FULL_V2 + i), NG); mbar_init(L::bar(L::B_EMPTY_V2 + i), NG);
    }
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  }
  tm_fence_before();
  __syncthreads();
  tm_fence_after();
  asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");   // the fills above precede the bulk copies

  const int role = warp >> 2, g = warp & 3;          // role 0..2 = A, B, C
  Ctx c;
  c.a = &s_args; c.xs = it.xs; c.plane = p; c.lane = lane; c.g = g; c.t = g * 32 + lane; c.nb = it.nb;
  c.flp = a.flags + it.fl_off + (g < NG ? g : 0);
  c.tm = s_tmem + ((uint32_t)(g * 32) << 16);
  const int x = it.xs + PX * c.t;                     // image column of the thread's first pixel
  const bool col_in = PX * c.t < a.CW && x < a.Dx;    // (Dx - xs) is a multiple of 8: a thread never straddles the image edge
  c.sx = col_in ? a.Dx : 0;
  const bool worker = g < NG;
  if (worker && role < 2) {     // zero the rings: group A the F ring, group B the d ring
    const float2 z[4] = {splat(0.f), splat(0.f), splat(0.f), splat(0.f)};
    for (int i = 0; i < DR; ++i) tm_st8(c.tm + (role ? TM_D : 0) + PX * i, z);
    tm_wait_st();
  }
  tm_fence_before();
  __syncthreads();
  tm_fence_after();

  const long long N = (long long)a.Dy * a.Dx;
  const float* X = (p < a.B) ? a.cube + (long long)p * N : a.sum_plane;
  if (worker) {
    if (role == 0) {
      RoleA<NG> r(c, a);
      r.dirty = *a.dirty == a.dirty_seq;
      r.y0 = it.y_start;
      r.producer = g == 0 && lane == 0;
      r.ys = it.y_start;
      {   // copied columns: the strip with 4 columns of margin, clipped to the image
        const int cx0 = it.xs - 4 > 0 ? it.xs - 4 : 0;
        const int cx1 = it.xs + a.CW + 4 < a.Dx ? it.xs + a.CW + 4 : a.Dx;
        r.row_bytes = (uint32_t)(cx1 - cx0) * 4u;
        r.xrow0 = X + (long long)it.y_start * a.Dx + cx0;
        r.x_dst0 = smem_u32(reinterpret_cast<const float*>(g_sm4) + L::O_X + (cx0 - (it.xs - 4)));
      }
      r.nmp = col_in ? a.nm_pad + (long long)(it.y_start - 3 + PADR) * a.Dx + x : a.nm_pad;   // lanes outside the strip read a zero row
#pragma unroll
      for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int q = 0; q < 4; ++q) r.hw[i][q] = splat(0.f);
#pragma unroll
      for (int q = 0; q < 4; ++q) r.V1[q] = splat(0.f);
#pragma unroll
      for (int j = 0; j < RB; ++j) { r.nm[j][0] = zero4(); r.nm[j][1] = zero4(); }
      r.run();
    } else if (role == 1) {
      RoleB<NG> r(c, a);
      r.icp = col_in ? a.ic_pad + (long long)(it.y_start - LAG_B + PADR) * a.Dx + x : a.nm_pad;
#pragma unroll
      for (int q = 0; q < 4; ++q) { r.V2[q] = splat(0.f); r.E[q] = splat(0.f); }
#pragma unroll
      for (int j = 0; j < RB; ++j) { r.ic[j][0] = zero4(); r.ic[j][1] = zero4(); }
      r.fr = 0;
      r.fq = 30;                // rho0 - 2 of step 0, modulo the 32 rows of the flag ring
#pragma unroll
      for (int i = 0; i < 6; ++i)
#pragma unroll
        for (int q = 0; q < 4; ++q) r.Fw[i][q] = splat(__int_as_float(0xff800000));
      r.run();
    } else {
      RoleC<NG> r(c, a);
      r.icp = col_in ? a.ic_pad + (long long)(it.y_start - LAG_C + PADR) * a.Dx + x : a.nm_pad;
#pragma unroll
      for (int j = 0; j < RB; ++j) { r.ic[j][0] = zero4(); r.ic[j][1] = zero4(); }
      r.fr = DF - KBG;          // sigma = rho - 12 of the same step
      r.y0 = it.y_start;
      r.umask = 0u;
#pragma unroll
      for (int k = 0; k < PX; ++k)
        if (col_in && x + k >= it.ux0 && x + k < it.ux1) r.umask |= 1u << k;
      r.run();
    }
  }

  tm_wait_st();
  tm_fence_before();
  __syncthreads();
  if (warp == 0)
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;\n" ::"r"(s_tmem), "n"(512));
}

}  // namespace

// ------------------------------------------------------------------------------------------------
// Work plan (host, once per context): column strips over the valid bounding box, row segments,
// the per-(step, warp column) control words of every item, zero-padded normaliser planes.
struct LpfFusedPlan {
  bool ok = false;
  int CW = 0, NG = 0, threads = 0, n_items = 0;
  size_t smem = 0;
  float nm_const = 1.f, ic_const = 1.f / 625.f;
  FusedItem* d_items = nullptr;
  uint32_t* d_flags = nullptr;
  float* d_nm_pad = nullptr;
  float* d_ic_pad = nullptr;
};

template <int NG>
static cudaError_t sweep_launch_t(const FusedArgs& a, dim3 grid, cudaStream_t st, bool set_attr, size_t* smem_out) {
  const size_t smem = (size_t)Lay<NG>::O_END * sizeof(float) + 16;
  if (smem_out) *smem_out = smem;
  if (set_attr) return cudaFuncSetAttribute(k_sweep_box<NG>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  k_sweep_box<NG><<<grid, NTHREADS, smem, st>>>(a);
  return cudaSuccess;
}

static cudaError_t sweep_dispatch(int NG, const FusedArgs& a, dim3 grid, cudaStream_t st, bool set_attr, size_t* smem_out) {
  switch (NG) {
    case 1: return sweep_launch_t<1>(a, grid, st, set_attr, smem_out);
    case 2: return sweep_launch_t<2>(a, grid, st, set_attr, smem_out);
    default: return sweep_launch_t<4>(a, grid, st, set_attr, smem_out);
  }
}

// class bits of a (row, warp column) cell of a strip
enum { CL_ANYW = 1,    // some valid pixel among the warp's columns +-4
       CL_NM1 = 4,     // norm_mf is the interior constant on all the warp's columns
       CL_IC1 = 8 };   // 1/count is 1/625 on all the warp's columns

int lpf_fused_plan(lpf_ctx* c, const uint8_t* hW, LpfFusedPlan** out) {
  *out = nullptr;
  const lpf_params& p = c->p;
  if (p.force_general) return LPF_OK;
  if (!(p.bg_kernel == 1 && p.k_bg == KBG && p.k_mf == 3 && p.sigma_mf > 0 && p.n_iter == 1 && (p.Dx % 8) == 0 &&
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
    const int uw = ((width + s - 1) / s + 7) / 8 * 8;
    strips.clear();
    int cw = 0;
    for (int i = 0; i < s; ++i) {
      FusedItem it{};
      it.ux0 = vx0 + i * uw; it.ux1 = std::min(vx1, it.ux0 + uw);
      if (it.ux0 >= it.ux1) continue;
      const int lo = std::max(vx0, it.ux0 - HALO), hi = std::min(vx1, it.ux1 + HALO);
      it.xs = lo / 8 * 8;
      const int xe = std::min(Dx, (hi + 7) / 8 * 8);
      cw = std::max(cw, xe - it.xs);
      strips.push_back(it);
    }
    if (cw <= 4 * GW) { n_strips = (int)strips.size(); CW = cw; }
  }
  if (!n_strips) return LPF_OK;
  int NG = 1;
  while (NG * GW < CW) NG *= 2;
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
  const int sm_share = std::max(1, c->n_sm / std::max(1, std::min(p.n_lanes, 4)));   // (more lanes in flight only deepen the queue)
  const double warm = (double)(HALO + 2 * RB * NV + 12);   // warm-up rows of a segment + the fill / drain of the rings
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
  // (row, warp column) classes of every strip, rows -CPAD .. Dy+CPAD
  const int CPAD = 128;
  std::vector<std::vector<uint8_t>> cls(strips.size());
  long long interior_pix = -1;
  for (size_t si = 0; si < strips.size(); ++si) {
    const int xs = strips[si].xs;
    cls[si].assign((size_t)(Dy + 2 * CPAD) * NG, 0);
    for (int y = 0; y < Dy; ++y)
      for (int w = 0; w < NG; ++w) {
        const int c0 = xs + GW * w, c1 = std::min(c0 + GW, xs + CW);   // own columns [c0, c1)
        if (c0 >= xs + CW) continue;
        int any = 0, nm1 = 1, ic1 = 1;
        for (int x = c0 - 4; x < c0 + GW + 4; ++x) {
          const bool in = x >= 0 && x < Dx && x >= xs - 4 && x < xs + CW + 4;
          any |= (in && hW[(size_t)y * Dx + x]) ? 1 : 0;
        }
        for (int x = c0; x < c0 + GW; ++x) {
          if (x >= c1) { nm1 = 0; ic1 = 0; break; }
          if (!full_window(y, x, 3)) nm1 = 0;
          if (!full_window(y, x, KBG)) ic1 = 0;
          if (!nm1 && !ic1) break;
        }
        if (nm1 && interior_pix < 0) interior_pix = (long long)y * Dx + c0;
        cls[si][(size_t)(y + CPAD) * NG + w] = (uint8_t)((any ? CL_ANYW : 0) | (nm1 ? CL_NM1 : 0) | (ic1 ? CL_IC1 : 0));
      }
  }
  // control words
  std::vector<uint32_t> flags;
  std::vector<FusedItem> ditems;
  for (auto& ie : items) {
    FusedItem it = ie.it;
    const std::vector<uint8_t>& cl = cls[ie.strip];
    auto cell = [&](int y, int w) -> int { return (y < -CPAD || y >= Dy + CPAD) ? 0 : cl[(size_t)(y + CPAD) * NG + w]; };
    int ys = it.ya - HALO;
    if (ys & 1) ys -= 1;               // even first row: a row pair never straddles the image edge (Dy is even)
    it.y_start = ys;
    it.nb = (it.yb - 1 + LAG_C - ys) / RB + 1;
    it.fl_off = (int)flags.size();
    auto xmode = [&](int y, int w) -> unsigned { return ((cell(y, w) | cell(y + 1, w)) & CL_ANYW) ? FL_X : 0u; };
    auto both = [&](int y, int w, int bit) -> bool { return (cell(y, w) & cell(y + 1, w) & bit) != 0; };
    for (int b = 0; b < it.nb; ++b)
      for (int w = 0; w < NG; ++w) {
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
        if (y0 + 1 - LAG_B >= it.ya - KBG - 2) f |= FL_DO_B;     // (two more rows: the local-maximum window of the first output row)
        if (y0 - LAG_C >= it.ya && y0 - LAG_C < it.yb) f |= FL_C0;
        if (y0 + 1 - LAG_C >= it.ya && y0 + 1 - LAG_C < it.yb) f |= FL_C1;
        flags.push_back(f);
      }
    ditems.push_back(it);
  }
  static_assert((FL_NM_LD << 3) == FL_NM_PF && (FL_ICR_LD << 3) == FL_ICR_PF && (FL_ICS_LD << 3) == FL_ICS_PF, "flag layout");

  LpfFusedPlan* pl = new LpfFusedPlan();
  pl->CW = CW; pl->NG = NG; pl->threads = NTHREADS; pl->n_items = (int)ditems.size();
  FusedArgs dummy{};
  *out = pl;   // owned by the context from here on (freed by lpf_destroy on any later failure)
  LPF_CUDA(sweep_dispatch(NG, dummy, dim3(1), 0, true, &pl->smem));
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
                            lpf_det* d_dets, int32_t* d_ndets, bool sum_done, cudaStream_t st) {
  const lpf_params& p = c->p;
  if (!sum_done) {     // the chained frame call has done both in its second QC pass
    LPF_CUDA(cudaMemsetAsync(d_ndets, 0, sizeof(int32_t), st));
    int rc = lpf_launch_sum_plane(c, L, d_cube, d_band_ok, p.detect_sum_plane != 0, st);   // + the exact-zero check
    if (rc) return rc;
  }
  FusedArgs a{};
  a.cube = d_cube; a.sum_plane = L.sum_plane; a.band_ok = d_band_ok; a.W = c->W;
  a.nm_pad = pl->d_nm_pad; a.ic_pad = pl->d_ic_pad; a.items = pl->d_items; a.flags = pl->d_flags; a.dirty = L.dirty; a.dirty_seq = L.dirty_seq;
  a.B = p.B; a.Dy = p.Dy; a.Dx = p.Dx; a.CW = pl->CW; a.k_max = p.k_max; a.max_det = p.max_det;
  a.g0 = c->g_mf.g[3]; a.g1 = c->g_mf.g[2]; a.g2 = c->g_mf.g[1]; a.g3 = c->g_mf.g[0];
  a.kappa2 = p.kappa * p.kappa; a.eps_rel = p.eps_rel; a.nm_const = pl->nm_const; a.ic_const = pl->ic_const;
  a.dets = d_dets; a.ndets = d_ndets; a.counters = c->counters;
  const dim3 grid(pl->n_items, c->n_planes);
  LPF_KLAUNCH(c, KID_FUSED_DETECT, st, sweep_dispatch(pl->NG, a, grid, st, false, nullptr));
  return LPF_OK;
}
