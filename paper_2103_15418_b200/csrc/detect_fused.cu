// S4-S8 fused fast path: matched filter -> local centre -> local spread -> sigma clip -> local
// maxima -> compaction in ONE pass over each plane, for the headline parameter set
// (box background K = 12, Gaussian matched filter k_mf = 3, n_iter = 1).
// (eqs. 2-7; O3-O6 and "Fused detection kernel".)
//
// Design (sm_100a).  A CTA owns a column strip (4 columns per thread, up to 1024 columns) and sweeps
// down a segment of rows, two rows per iteration, as a three-stage software pipeline with ONE
// block barrier per iteration (the stages of one iteration work on different rows, so their
// shared-memory exchanges are double buffered and independent):
//   A  rows y:        the input rows arrive in shared memory by bulk asynchronous copies (TMA,
//                     cp.async.bulk + mbarrier) issued three iterations ahead by one thread; every
//                     thread reads its 4 pixels and both neighbours' with three 128-bit shared loads ->
//                     horizontal 7-tap matched filter -> vertical 7-tap on a register window (packed
//                     f32x2) -> F(y-3); 25-row running sum V1 += F(y-3) - F(y-28)
//   B  rows rho=y-17: horizontal 25-box of V1 (blocked partial sums) x 1/count -> C (eq. 3);
//                     d = F - C; 25-row running sum V2 += d^2 - d_old^2
//   C  rows sig=y-31: horizontal 25-box of V2 x 1/count -> S (eq. 4); eq. 5 on d(sig) for the whole
//                     row with four packed operations and one vote; rows with a hit go out of line:
//                     exact bits, a cheap in-thread 3x3 pre-filter on the F ring, then the S_eff guard
//                     (R8), eq. 6 with one neighbour per lane and the eq. 7 record.
// The 32-row histories of F and d that the running sums and the lagged reads need are private to
// a thread, so they live in TENSOR MEMORY (tcgen05.st/ld 32x32b.x4, two power-of-two rings of 128
// columns per thread); shared memory carries only what threads exchange plus a 32-row ring of F for
// the local-maximum tests.  What a warp has to decide in an iteration (is there input, which
// normalisers are the interior constants, which stages run) is one 32-bit word of a per-item table
// built by the host plan.  F, C, d, S never leave the SM.
// The input is used unmasked when the cube holds exact zeros at every invalid pixel (checked per
// frame by the sum-plane kernel); otherwise each thread applies W itself (slow, rare).
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
constexpr int DRS = 34;             // depth of the shared-memory ring of F: local maxima are tested one iteration late
constexpr int QCAP = 64;            // queued candidates per iteration (more are tested in place)
constexpr int SCAP = 32;            // records staged by a helper warp between flushes
constexpr int NHW = 3;              // helper warps: input producer and candidate tests
constexpr int XST = 4;              // input staging stages (iterations in flight)
constexpr int TM_D = 4 * DR;        // first tensor-memory column of the d ring (F ring starts at 0)
constexpr int PADR = 64;            // zero rows above and below the padded normaliser planes

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

// ---- candidate path ---------------------------------------------------------------------------------
// Pixels that pass the unguarded eq. 5 are queued by the sweep warps (a few per iteration) and tested one
// iteration later by a dedicated warp, off the sweep's critical path: S_eff guard (R8), eq. 6 on the
// shared-memory ring of F, eq. 7 record.  One candidate per lane, up to 32 at a time.
struct CandCtx {           // what the candidate functions need, by value
  const FusedArgs* ap;     // kernel arguments (shared-memory copy)
  int CWP, xs, plane, lane, ring_y0;
};

__device__ __forceinline__ int ring_slot(int row, int ring_y0) { return (int)((unsigned)(row - ring_y0) % (unsigned)DRS); }

// the test of one candidate by its own lane; returns true when it is a peak (fills f, c, s_eff).
// KM = k_max at compile time (fully unrolled window, independent shared loads); KM < 0: run-time k_max.
template <int KM>
__device__ __forceinline__ bool cand_test_lane(const CandCtx& c, int cl, int sg, float d, float s,
                                               float& fv, float& cc, float& se) {
  const FusedArgs& a = *c.ap;
  const int CWP = c.CWP;
  const int s0 = ring_slot(sg, c.ring_y0);
  fv = lds1(s0 * CWP + cl);
  cc = fv - d;
  const float gd = a.eps_rel * fabsf(cc);
  se = fmaxf(s, gd * gd);
  if (!(d > 0.f && d * d > a.kappa2 * se)) return false;
  const int km = KM >= 0 ? KM : a.k_max;
  bool bigger = false, zero_wins = false;       // a neighbour with F = 0 > fv: masked or not?  (rare: asks W)
#pragma unroll
  for (int dy = -km; dy <= km; ++dy) {
    const int yy = sg + dy;
    int sl = s0 + dy;
    sl = sl < 0 ? sl + DRS : (sl >= DRS ? sl - DRS : sl);
    const bool row_in = yy >= 0 && yy < a.Dy;
#pragma unroll
    for (int dx = -km; dx <= km; ++dx) {
      const int c2 = cl + dx;
      const bool in = row_in && c2 >= 0 && c2 < CWP && c.xs + c2 < a.Dx;
      const float fn = in ? lds1(sl * CWP + c2) : fv;
      bigger = bigger || (fn > fv && fn != 0.f);
      zero_wins = zero_wins || (fn > fv && fn == 0.f);
    }
  }
  if (bigger) return false;
  if (zero_wins) {
    for (int dy = -km; dy <= km; ++dy)
      for (int dx = -km; dx <= km; ++dx) {
        const int yy = sg + dy, c2 = cl + dx, xn = c.xs + c2;
        if (yy < 0 || yy >= a.Dy || c2 < 0 || c2 >= CWP || xn >= a.Dx) continue;
        if (lds1(ring_slot(yy, c.ring_y0) * CWP + c2) > fv && a.W[(long long)yy * a.Dx + xn] != 0) return false;
      }
  }
  return true;
}

__device__ __forceinline__ bool cand_test_any(const CandCtx& c, int cl, int sg, float d, float s, float& fv, float& cc, float& se) {
  const int km = c.ap->k_max;
  if (km == 2) return cand_test_lane<2>(c, cl, sg, d, s, fv, cc, se);
  if (km == 1) return cand_test_lane<1>(c, cl, sg, d, s, fv, cc, se);
  return cand_test_lane<-1>(c, cl, sg, d, s, fv, cc, se);
}

// staged records (shared memory, 8 words each, n of them at float index o_st) -> global list, one atomic
__device__ __noinline__ void cand_flush(const FusedArgs* ap, int o_st, int lane, int n) {
  if (n <= 0) return;
  int base = 0;
  if (lane == 0) base = atomicAdd(ap->ndets, n);
  base = __shfl_sync(0xffffffffu, base, 0);
  for (int i = lane; i < n; i += 32) {
    const uint2* r = reinterpret_cast<const uint2*>(reinterpret_cast<const uint32_t*>(g_sm4) + o_st + i * 8);
    const int idx = base + i;
    if (idx < ap->max_det) {
      uint2* dst = reinterpret_cast<uint2*>(ap->dets + idx);
      uint2 r2 = r[2];
      r2.y = __float_as_uint(__uint_as_float(r2.y) / sqrtf(__uint_as_float(r2.x)));
      dst[0] = r[0]; dst[1] = r[1]; dst[2] = r2;
    } else {
      atomicAdd(&ap->counters[0], 1);
    }
  }
  __syncwarp();
}

// lanes with ok stage their records at o_st (nst staged so far, room for SCAP); returns the new count
__device__ __forceinline__ int cand_stage(const CandCtx& c, int o_st, int nst, bool ok, int cl, int sg, float d, float fv, float cc, float se) {
  const FusedArgs& a = *c.ap;
  const unsigned m = __ballot_sync(0xffffffffu, ok);
  if (!m) return nst;
  if (nst + __popc(m) > SCAP) { cand_flush(c.ap, o_st, c.lane, nst); nst = 0; }
  if (ok) {
    uint32_t* r = reinterpret_cast<uint32_t*>(g_sm4) + o_st + (nst + __popc(m & ((1u << c.lane) - 1u))) * 8;
    r[0] = (uint32_t)(sg * a.Dx + c.xs + cl);
    r[1] = (uint32_t)(c.plane & 0xffff) | (1u << 16);        // int16 plane, int16 iter = 1
    r[2] = __float_as_uint(fv); r[3] = __float_as_uint(cc); r[4] = __float_as_uint(se);
    r[5] = __float_as_uint(d);                               // snr = d / sqrt(s_eff) is taken at flush time
  }
  __syncwarp();
  return nst + __popc(m);
}

// k_max = 2: five lanes per candidate, one window row each (six candidates per warp and pass).  e0: the
// warp's first entry of this pass.  Queue entry: {col | slot << 16, row, d, s}, slot = the row's place in
// the F ring.  Written for a short dependent chain: all six shared loads leave together.
struct CandK { float kappa2, eps_rel; int Dy, Dx; const uint8_t* W; };
__device__ __forceinline__ int cand_pass5(const CandCtx& c, const CandK& k, int o_q, int n, int e0, int o_st, int nst) {
  const int CWP = c.CWP;
  const int g = (c.lane * 13) >> 6, r = c.lane - 5 * g;        // lane / 5, lane % 5 (lanes 30, 31: g = 6, idle)
  const int e = e0 + g;
  const bool act = g < 6 && e < n;
  const float4 q = lds4(o_q + 4 * (act ? e : 0));
  const int cs = __float_as_int(q.x), cl = cs & 0xffff, s0 = cs >> 16, sg = __float_as_int(q.y);
  const float d = q.z;
  int sl = s0 + r - 2;
  sl = sl < 0 ? sl + DRS : (sl >= DRS ? sl - DRS : sl);
  const int yy = sg + r - 2;
  const int rb = sl * CWP;
  const float fv = lds1(s0 * CWP + cl);
  float fn[5];
#pragma unroll
  for (int dx = 0; dx < 5; ++dx) {
    int c2 = cl + dx - 2;
    c2 = c2 < 0 ? 0 : (c2 >= CWP ? CWP - 1 : c2);
    fn[dx] = lds1(rb + c2);
  }
  const float cc = fv - d;
  const float gd = k.eps_rel * fabsf(cc);
  const float se = fmaxf(q.w, gd * gd);
  const bool pass = act && d > 0.f && d * d > k.kappa2 * se;
  const bool row_in = pass && yy >= 0 && yy < k.Dy;
  bool bigger = false;
#pragma unroll
  for (int dx = 0; dx < 5; ++dx) {
    const int c2 = cl + dx - 2, xn = c.xs + c2;
    const bool in = row_in && c2 >= 0 && c2 < CWP && xn < k.Dx;
    // masked pixels hold F = 0 in the ring: W is consulted only when such a zero would win
    if (in && fn[dx] > fv) bigger = bigger || (fn[dx] != 0.f) || (k.W[(long long)yy * k.Dx + xn] != 0);
  }
  const unsigned ball = __ballot_sync(0xffffffffu, bigger);
  const bool ok = pass && r == 0 && ((ball >> (5 * g)) & 31u) == 0u;
  return cand_stage(c, o_st, nst, ok, cl, sg, d, fv, cc, se);
}

// the queue of one iteration, n entries {col, row, d, s} at float index o_q: the share of helper warp hw of nh
__device__ __noinline__ int cand_consume(CandCtx c, int o_q, int n, int hw, int nh, int o_st, int nst) {
  for (int e0 = 32 * hw; e0 < n; e0 += 32 * nh) {
    const int e = e0 + c.lane;
    bool ok = false;
    int cl = 0, sg = 0; float d = 0.f, fv = 0.f, cc = 0.f, se = 1.f;
    if (e < n) {
      const float4 q = lds4(o_q + 4 * e);
      cl = __float_as_int(q.x) & 0xffff; sg = __float_as_int(q.y); d = q.z;
      ok = cand_test_any(c, cl, sg, d, q.w, fv, cc, se);
    }
    nst = cand_stage(c, o_st, nst, ok, cl, sg, d, fv, cc, se);
  }
  return nst;
}

// a sweep warp whose candidates did not fit the queue (rare: a row full of bright pixels) tests them itself
// and appends the records straight to the global list
__device__ __noinline__ void cand_in_place(CandCtx c, unsigned bits, int col0, int sg, float4 dv, float4 sv) {
  const FusedArgs& a = *c.ap;
  const float d[4] = {dv.x, dv.y, dv.z, dv.w};
  const float s[4] = {sv.x, sv.y, sv.z, sv.w};
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    float fv = 0.f, cc = 0.f, se = 1.f;
    bool ok = false;
    if ((bits >> k) & 1u) ok = cand_test_lane<-1>(c, col0 + k, sg, d[k], s[k], fv, cc, se);
    const unsigned m = __ballot_sync(0xffffffffu, ok);
    if (!m) continue;
    int base = 0;
    if (c.lane == 0) base = atomicAdd(a.ndets, __popc(m));
    base = __shfl_sync(0xffffffffu, base, 0);
    if (ok) {
      const int idx = base + __popc(m & ((1u << c.lane) - 1u));
      if (idx < a.max_det) {
        uint2* dst = reinterpret_cast<uint2*>(a.dets + idx);
        dst[0] = make_uint2((uint32_t)(sg * a.Dx + c.xs + col0 + k), (uint32_t)(c.plane & 0xffff) | (1u << 16));
        dst[1] = make_uint2(__float_as_uint(fv), __float_as_uint(cc));
        dst[2] = make_uint2(__float_as_uint(se), __float_as_uint(d[k] / sqrtf(se)));
      } else {
        atomicAdd(&a.counters[0], 1);
      }
    }
  }
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

template <int NW>
struct Sweep {
  static constexpr int CWP = NW * 128;             // shared-memory row pitch: the CTA's full width
  static constexpr int XP = CWP + 8;               // staged input row: 4 columns of margin on both sides
  static constexpr int PEV = CWP + 2 * KBG, PET = NW * 32 + 8;
  static constexpr int O_RING = 0;
  static constexpr int O_X = DRS * CWP;
  static constexpr int O_EV1 = O_X + XST * RB * XP;
  static constexpr int O_EV2 = O_EV1 + 2 * RB * PEV;
  static constexpr int O_ET1 = O_EV2 + 2 * RB * PEV;
  static constexpr int O_ET2 = O_ET1 + 2 * RB * PET;
  static constexpr int O_Q = O_ET2 + 2 * RB * PET;       // candidate queues, [2][QCAP] x {col, row, d, s}
  static constexpr int O_QN = O_Q + 2 * QCAP * 4;        // their lengths, one word per iteration mod 4
  static constexpr int O_ST = O_QN + 4;                  // staged records of the helper warps, [NHW][SCAP] x 8 words
  static constexpr int O_BAR = O_ST + NHW * SCAP * 8;    // XST mbarriers (8 bytes each)
  static constexpr int O_FL = O_BAR + 2 * XST + 2;       // end of the layout (XST input barriers + the iteration barrier)
  // ---- constants of the thread -----------------------------------------------------------------
  const FusedArgs& a;
  const FusedArgs* a_sh;   // the same arguments in shared memory (for the out-of-line candidate path)
  int xs, plane, tid, lane, warp;
  const uint32_t* flp;     // this warp's control words, [nb] with stride NW
  int sx;                  // row stride of the plane pointers (0 for lanes outside the strip)
  bool col_in, dirty;
  unsigned umask;
  uint32_t tm;             // tensor-memory address of the thread's column 0
  // producer (thread 0)
  const float* xrow0;      // X at (y_start, first copied column)
  uint32_t x_dst0;         // shared address of that column in stage 0, row 0
  uint32_t row_bytes;
  int nb;
  // ---- running state -----------------------------------------------------------------------------
  const float* nmp;        // padded norm_mf at the next iteration's first F row
  const float* icrp;       // padded 1/count at the next iteration's first rho row
  const float* icsp;       // padded 1/count at the next iteration's first sigma row
  int y0;                  // first input row of the current iteration
  int ring_y0;             // the row that sits in slot 0 of the rings
  int ws;                  // slot of this iteration's first F row in the shared-memory ring
  float2 hw[8][2];         // horizontally filtered rows (rotating; static indices per phase)
  float2 V1[2], V2[2];     // vertical running sums
  Planes pl;               // normalisers of the coming rows: each plane is reloaded right after its use

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

  // the per-iteration barrier of all warps, in two halves (an mbarrier with one arrival per warp: 32 arrivals on
  // one shared-memory word would serialise)
  __device__ __forceinline__ void sync_arrive() const { __syncwarp(); if (lane == 0) mbar_arrive(bar_addr(XST)); }
  __device__ __forceinline__ void sync_wait(int b) const { mbar_wait(bar_addr(XST), (uint32_t)b & 1u); }

  __device__ __forceinline__ CandCtx cand_ctx() const {
    CandCtx c;
    c.ap = a_sh; c.CWP = CWP; c.xs = xs; c.plane = plane; c.lane = lane; c.ring_y0 = ring_y0;
    return c;
  }

  // thread 0: the two input rows of iteration bb into stage bb mod XST (a plain arrival when they lie outside the image)
  __device__ __forceinline__ void issue_rows(int bb, int ys) {
    const int st = bb & (XST - 1);
    const uint32_t bar = bar_addr(st);
    const int y = ys + RB * bb;
    if (bb >= XST) mbar_wait(bar, (uint32_t)((bb >> 2) - 1) & 1u);   // its previous phase (complete unless no warp waited for it)
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

  __device__ __forceinline__ void load_nm(unsigned on) {
    if (on) { pl.nm[0] = ldg4_pinned(nmp); pl.nm[1] = ldg4_pinned(nmp + sx); }
    nmp += RB * sx;
  }
  __device__ __forceinline__ void load_icr(unsigned on) {
    if (on) { pl.icr[0] = ldg4_pinned(icrp); pl.icr[1] = ldg4_pinned(icrp + sx); }
    icrp += RB * sx;
  }
  __device__ __forceinline__ void load_ics(unsigned on) {
    if (on) { pl.ics[0] = ldg4_pinned(icsp); pl.ics[1] = ldg4_pinned(icsp + sx); }
    icsp += RB * sx;
  }

  // Stage A, part 1 for iteration bn (PH = bn mod 4): staged input rows -> horizontal matched filter -> hw.
  // It touches only the input stages and registers, so it runs in the shadow of the previous iteration's
  // barrier (between the arrival and the wait).  yn: first input row of iteration bn.
  template <int PH>
  __device__ __forceinline__ void stage_a1(int bn, unsigned fl, int yn) {
    if (fl & FL_X) {
      mbar_wait(bar_addr(PH), (uint32_t)(bn >> 2) & 1u);
#pragma unroll
      for (int j = 0; j < RB; ++j) {
        const int xr = O_X + (PH * RB + j) * XP + 4 * tid;
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
        hw[(2 * PH + 6 + j) & 7][0] = make_float2(h[0], h[1]);
        hw[(2 * PH + 6 + j) & 7][1] = make_float2(h[2], h[3]);
      }
    } else {
#pragma unroll
      for (int j = 0; j < RB; ++j) { hw[(2 * PH + 6 + j) & 7][0] = splat(0.f); hw[(2 * PH + 6 + j) & 7][1] = splat(0.f); }
    }

  }

  // One iteration: rows y0, y0+1 enter stage A; PH = iteration index mod 4 fixes the register rotation
  // and the staging stage.  fl: this iteration's control word.
  template <int PH>
  __device__ __forceinline__ void iteration(int b, unsigned fl, unsigned fl_next) {
    constexpr int buf = PH & 1, pbuf = buf ^ 1;
    const float2 g0 = splat(a.g0), g1 = splat(a.g1), g2 = splat(a.g2), g3 = splat(a.g3);
    const int w = (RB * b) & (DR - 1);                       // ring slot of this iteration's first row (even)
    const uint32_t t_old0 = tm + 4u * (uint32_t)((w + 7) & (DR - 1)), t_old1 = tm + 4u * (uint32_t)((w + 8) & (DR - 1));
    const uint32_t t_lag0 = tm + 4u * (uint32_t)((w + 18) & (DR - 1)), t_lag1 = t_lag0 + 4u;   // w + 18 is even: no wrap in between
    const uint32_t t_new0 = tm + 4u * (uint32_t)w, t_new1 = t_new0 + 4u;

    // ---- tensor-memory reads: F(fr - 25), F(rho), d(rho - 25), d(sigma) ---------------------------------
    float2 fold[RB][2], flag[RB][2], dold[RB][2], dlag[RB][2];
    tm_ld4(t_old0, fold[0][0], fold[0][1]); tm_ld4(t_old1, fold[1][0], fold[1][1]);


    tm_wait_ld();
#pragma unroll
    for (int j = 0; j < RB; ++j) tm_use(fold[j][0], fold[j][1]);
    // second batch, for stages B and C: F(rho), d(rho - 25), d(sigma)
    tm_ld4(t_lag0, flag[0][0], flag[0][1]); tm_ld4(t_lag1, flag[1][0], flag[1][1]);
    tm_ld4(t_old0 + TM_D, dold[0][0], dold[0][1]); tm_ld4(t_old1 + TM_D, dold[1][0], dold[1][1]);
    tm_ld4(t_lag0 + TM_D, dlag[0][0], dlag[0][1]); tm_ld4(t_lag1 + TM_D, dlag[1][0], dlag[1][1]);

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
          f[j][0] = mul2(f[j][0], make_float2(pl.nm[j].x, pl.nm[j].y));
          f[j][1] = mul2(f[j][1], make_float2(pl.nm[j].z, pl.nm[j].w));
        }
      } else {
        const float2 c = splat(a.nm_const);
#pragma unroll
        for (int j = 0; j < RB; ++j) { f[j][0] = mul2(f[j][0], c); f[j][1] = mul2(f[j][1], c); }
      }
#pragma unroll
      for (int j = 0; j < RB; ++j) {
        V1[0] = add2(V1[0], sub2(f[j][0], fold[j][0]));
        V1[1] = add2(V1[1], sub2(f[j][1], fold[j][1]));
        tm_st4(j ? t_new1 : t_new0, f[j][0], f[j][1]);
        sts4(O_RING + (ws + j) * CWP + 4 * tid, make_float4(f[j][0].x, f[j][0].y, f[j][1].x, f[j][1].y));
        sts4(O_EV1 + (buf * RB + j) * PEV + KBG + 4 * tid, make_float4(V1[0].x, V1[0].y, V1[1].x, V1[1].y));
        const float2 ts = add2(V1[0], V1[1]);
        sts1(O_ET1 + (buf * RB + j) * PET + 3 + tid, ts.x + ts.y);
      }
    }

    load_nm(fl & FL_NM_PF);                          // the next iteration's norm_mf rows
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
        if (fl & FL_ICR_LD) { ic0 = make_float2(pl.icr[j].x, pl.icr[j].y); ic1 = make_float2(pl.icr[j].z, pl.icr[j].w); }
        else { ic0 = splat(a.ic_const); ic1 = ic0; }
        dd[j][0] = fma2(make_float2(-bx[0], -bx[1]), ic0, flag[j][0]);     // d = F - box * (1/count)
        dd[j][1] = fma2(make_float2(-bx[2], -bx[3]), ic1, flag[j][1]);
      }
#pragma unroll
      for (int j = 0; j < RB; ++j) {
        V2[0] = fma2(neg2(dold[j][0]), dold[j][0], fma2(dd[j][0], dd[j][0], V2[0]));
        V2[1] = fma2(neg2(dold[j][1]), dold[j][1], fma2(dd[j][1], dd[j][1], V2[1]));
        tm_st4((j ? t_new1 : t_new0) + TM_D, dd[j][0], dd[j][1]);
        sts4(O_EV2 + (buf * RB + j) * PEV + KBG + 4 * tid, make_float4(V2[0].x, V2[0].y, V2[1].x, V2[1].y));
        const float2 ts = add2(V2[0], V2[1]);
        sts1(O_ET2 + (buf * RB + j) * PET + 3 + tid, ts.x + ts.y);
      }
    }

    load_icr(fl & FL_ICR_PF);

    // ---- stage C: S = box(V2) / count at sigma ; eq. 5 for the row ; candidates ------------------------
    if (fl & (FL_C0 | FL_C1)) {
#pragma unroll
      for (int j = 0; j < RB; ++j) {
        if (!(fl & (FL_C0 << j))) continue;          // uniform
        float bx[4];
        hbox25(O_EV2 + (pbuf * RB + j) * PEV + 4 * tid, O_ET2 + (pbuf * RB + j) * PET + tid, bx);
        float2 ic0, ic1;
        if (fl & FL_ICS_LD) { ic0 = make_float2(pl.ics[j].x, pl.ics[j].y); ic1 = make_float2(pl.ics[j].z, pl.ics[j].w); }
        else { ic0 = splat(a.ic_const); ic1 = ic0; }
        const float2 s0 = mul2(make_float2(bx[0], bx[1]), ic0), s1 = mul2(make_float2(bx[2], bx[3]), ic1);
        const float2 k0 = mul2(s0, splat(a.kappa2)), k1 = mul2(s1, splat(a.kappa2));
        // d^2 - kappa^2 S > 0 somewhere in the warp's row?  (the sign of the difference is exact)
        const float2 m0 = fma2(dlag[j][0], dlag[j][0], neg2(k0)), m1 = fma2(dlag[j][1], dlag[j][1], neg2(k1));
        const float mm = fmaxf(fmaxf(m0.x, m0.y), fmaxf(m1.x, m1.y));
        if (__any_sync(0xffffffffu, mm > 0.f)) {
          // exact bits (the sign of m is that of d^2 - kappa^2 S), then the queue of this iteration
          const float dv[4] = {dlag[j][0].x, dlag[j][0].y, dlag[j][1].x, dlag[j][1].y};
          const float mv[4] = {m0.x, m0.y, m1.x, m1.y};
          unsigned bits = 0u;
#pragma unroll
          for (int k = 0; k < 4; ++k)
            if (dv[k] > 0.f && mv[k] > 0.f) bits |= 1u << k;
          bits &= umask;
          const float sv[4] = {s0.x, s0.y, s1.x, s1.y};
          const int sg = y0 + j - LAG_C;
          int sslot = ws + j - (LAG_C - 3);                    // ring slot of row sigma (this iteration's F row j: ws + j)
          sslot = sslot < 0 ? sslot + DRS : sslot;
          if (bits) {
            int pos = atomicAdd(reinterpret_cast<int*>(g_sm4) + O_QN + (b & 3), __popc(bits));
#pragma unroll
            for (int k = 0; k < 4; ++k)
              if (((bits >> k) & 1u) && pos < QCAP) {
                sts4(O_Q + (buf * QCAP + pos) * 4, make_float4(__int_as_float((4 * tid + k) | (sslot << 16)), __int_as_float(sg), dv[k], sv[k]));
                ++pos; bits &= ~(1u << k);
              }
          }
          if (__any_sync(0xffffffffu, bits != 0u))     // queue full
            cand_in_place(cand_ctx(), bits, 4 * tid, sg, make_float4(dv[0], dv[1], dv[2], dv[3]), make_float4(sv[0], sv[1], sv[2], sv[3]));
        }
      }
    }
    load_ics(fl & FL_ICS_PF);
    ws = ws + RB >= DRS ? ws + RB - DRS : ws + RB;
    y0 += RB;
    tm_wait_st();
    // split barrier: arrive, filter the next iteration's input rows while the slower warps finish, wait
    sync_arrive();
    stage_a1<(PH + 1) & 3>(b + 1, fl_next, y0);
    sync_wait(b);
  }

  // the helper warps: helper 0 feeds the input stages (bulk copies three iterations ahead); all of them test
  // what the sweep warps queued in the previous iteration.  Same barriers as run().
  __device__ __forceinline__ void run_helper(int ys) {
    int* qn = reinterpret_cast<int*>(g_sm4) + O_QN;
    const int hw = warp - NW;
    const int o_st = O_ST + hw * SCAP * 8;
    int nst = 0;
    const CandCtx cc = cand_ctx();
    CandK ck; ck.kappa2 = a.kappa2; ck.eps_rel = a.eps_rel; ck.Dy = a.Dy; ck.Dx = a.Dx; ck.W = a.W;
    const bool km2 = a.k_max == 2;
    for (int b = 0; b <= nb; ++b) {
      if (hw == NHW - 1 && lane == 0) {
        if (b + XST - 1 < nb) issue_rows(b + XST - 1, ys);     // their stage was read in iteration b - 1
        qn[(b + 1) & 3] = 0;                                   // next iteration's counter (last read in b - 2)
      }
      if (b > 0) {
        const int n = min(qn[(b - 1) & 3], QCAP);
        if (n > 0) {
          const int o_q = O_Q + ((b - 1) & 1) * QCAP * 4;
          if (km2) { for (int e0 = 6 * hw; e0 < n; e0 += 6 * NHW) nst = cand_pass5(cc, ck, o_q, n, e0, o_st, nst); }
          else nst = cand_consume(cc, o_q, n, hw, NHW, o_st, nst);
        }
      }
      if (b < nb) { sync_arrive(); sync_wait(b); }
    }
    cand_flush(a_sh, o_st, lane, nst);
    if (hw == NHW - 1 && lane == 0)                   // no bulk copy may be in flight when the CTA leaves
      for (int bb = nb > XST ? nb - XST : 0; bb < nb; ++bb) mbar_wait(bar_addr(bb & (XST - 1)), (uint32_t)(bb >> 2) & 1u);
  }

  __device__ __forceinline__ void run() {
    {
      const unsigned f0 = ctl(0);
      load_nm(f0 & FL_NM_LD); load_icr(f0 & FL_ICR_LD); load_ics(f0 & FL_ICS_LD);
    }
    int b = 0;
    unsigned f0 = ctl(0), f1 = ctl(1), f2 = ctl(2);
    stage_a1<0>(0, f0, y0);
    while (true) {
      unsigned f3 = ctl(b + 3);
      iteration<0>(b, f0, f1); if (++b >= nb) break;
      f0 = ctl(b + 3);
      iteration<1>(b, f1, f2); if (++b >= nb) break;
      f1 = ctl(b + 3);
      iteration<2>(b, f2, f3); if (++b >= nb) break;
      f2 = ctl(b + 3);
      iteration<3>(b, f3, f0); if (++b >= nb) break;
    }
  }
};

template <int NW>
__global__ void __launch_bounds__(NW * 32 + NHW * 32, 1)
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
  s.nb = it.nb;
  s.dirty = *a.dirty == a.dirty_seq;
  if (s.tid == 0) s_args = a;
  constexpr int NT = NW * 32 + NHW * 32;    // NW sweep warps and the helper warps
  for (int i = s.tid; i < (SW::O_FL >> 2); i += NT) g_sm4[i] = zero4();
  s.flp = a.flags + it.fl_off + (s.warp < NW ? s.warp : 0);
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
    mbar_init(s.bar_addr(XST), NT / 32);
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  }
  asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");   // the zero fill above precedes the bulk copies
  const uint32_t tm_base = s_tmem;
  // warp w reaches the 32 lanes (w mod 4) * 32 ...; warps w and w+4 share them on different columns
  s.tm = tm_base + ((uint32_t)((s.warp & 3) * 32) << 16) + (uint32_t)(s.warp >> 2) * 256u;
  const bool sweeper = s.warp < NW;
  if (sweeper) {
    for (int i = 0; i < 2 * DR; ++i) tm_st4(s.tm + 4 * i, splat(0.f), splat(0.f));
    tm_wait_st();
  }

  const long long N = (long long)a.Dy * a.Dx;
  const float* X = (p < a.B) ? a.cube + (long long)p * N : a.sum_plane;
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
    s.nmp = a.nm_pad + (long long)(it.y_start - 3 + PADR) * a.Dx + x;
    s.icrp = a.ic_pad + (long long)(it.y_start - LAG_B + PADR) * a.Dx + x;
    s.icsp = a.ic_pad + (long long)(it.y_start - LAG_C + PADR) * a.Dx + x;
  } else {              // lanes outside the strip read the zero row of a padded plane, over and over
    s.sx = 0;
    s.nmp = a.nm_pad; s.icrp = a.nm_pad; s.icsp = a.nm_pad;
  }
#pragma unroll
  for (int i = 0; i < 8; ++i) { s.hw[i][0] = splat(0.f); s.hw[i][1] = splat(0.f); }
  s.V1[0] = s.V1[1] = s.V2[0] = s.V2[1] = splat(0.f);
#pragma unroll
    for (int j = 0; j < RB; ++j) { s.pl.nm[j] = zero4(); s.pl.icr[j] = zero4(); s.pl.ics[j] = zero4(); }
  s.ring_y0 = it.y_start - 3; s.ws = 0;
  __syncthreads();
  if (s.tid == (NW + NHW - 1) * 32)
    for (int bb = 0; bb < XST - 1 && bb < it.nb; ++bb) s.issue_rows(bb, it.y_start);

  if (sweeper) s.run(); else s.run_helper(it.y_start);

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
  const int CWP = NW * 128, XP = CWP + 8, PEV = CWP + 2 * KBG, PET = NW * 32 + 8;
  const size_t nfl = (size_t)DRS * CWP + (size_t)XST * RB * XP + 4 * RB * PEV + 4 * RB * PET + 2 * QCAP * 4 + 4 + NHW * SCAP * 8 + 2 * XST + 2;
  (void)max_nb;                 // the control words stay in global memory
  return nfl * sizeof(float) + 16;
}

template <int NW>
static cudaError_t fused_launch_t(const FusedArgs& a, dim3 grid, size_t smem, cudaStream_t st, bool set_attr) {
  if (set_attr) return cudaFuncSetAttribute(k_fused_box<NW>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  k_fused_box<NW><<<grid, NW * 32 + NHW * 32, smem, st>>>(a);
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
  // segments per strip: minimise waves x (rows per segment + warm-up cost) over the segment count.  With
  // n_lanes frames in flight the kernels of different lanes share the SMs, so each gets its share of them
  // (fewer, longer segments: less warm-up per output row).
  const int n_planes = c->n_planes;
  const int sm_share = std::max(1, c->n_sm / std::max(1, std::min(p.n_lanes, 4)));   // (more lanes in flight only deepen the queue)
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
  pl->CW = CW; pl->NW = NW; pl->threads = NW * 32 + NHW * 32; pl->n_items = (int)ditems.size();
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
  LPF_KLAUNCH(c, KID_FUSED_DETECT, st, fused_dispatch(pl->NW, a, grid, pl->smem, st, false));
  return LPF_OK;
}
