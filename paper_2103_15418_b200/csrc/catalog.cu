// S9-S12: duplicate filter, association + monitoring, forced flux, dynamic-spectrum rings.
// (O7-O10.)  All integer / compare work: results are exact.
#include <math_constants.h>

#include <algorithm>

#include "lpf_internal.cuh"

namespace {

constexpr int CAT_BLOCKS = 64, CAT_THREADS = 256;
constexpr int SORT_CAP = 8192;      // unique positions ranked from shared memory (more: from global memory)

// key: larger snr wins, equal snr -> lower plane wins.  snr > 0 so its bit pattern is monotone.
__device__ __forceinline__ unsigned long long dd_key(float snr, int plane) {
  return ((unsigned long long)__float_as_uint(snr) << 32) | (unsigned)(0x7fff - plane);
}

__global__ void __launch_bounds__(CAT_THREADS)
k_dedupe_scatter(const lpf_det* __restrict__ dets, const int32_t* __restrict__ ndets, int max_det,
                 unsigned long long* __restrict__ M, int32_t* __restrict__ tmp_n) {
  const int n = min(*ndets, max_det);
  if (blockIdx.x == 0 && threadIdx.x == 0) *tmp_n = 0;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x)
    atomicMax(&M[dets[i].pix], dd_key(dets[i].snr, dets[i].plane));
}

__global__ void __launch_bounds__(CAT_THREADS)
k_dedupe_select(const lpf_det* __restrict__ dets, const int32_t* __restrict__ ndets, int max_det,
                const unsigned long long* __restrict__ M, int Dy, int Dx, int r,
                int32_t* __restrict__ tmp_pos, int16_t* __restrict__ tmp_plane, float* __restrict__ tmp_snr,
                int32_t* __restrict__ tmp_n) {
  const int n = min(*ndets, max_det);
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    const lpf_det d = dets[i];
    const unsigned long long key = dd_key(d.snr, d.plane);
    if (M[d.pix] != key) continue;  // not the best plane at this pixel
    const int y = d.pix / Dx, x = d.pix - y * Dx;
    bool keep = true;
    const unsigned si = (unsigned)(key >> 32);
    if (r <= 2) {                       // the usual radius: the 5x5 loads are independent and leave together
      unsigned long long kq[25];
#pragma unroll
      for (int j = -2; j <= 2; ++j)
#pragma unroll
        for (int k = -2; k <= 2; ++k) {
          const int yy = y + j, xx = x + k;
          const bool in = yy >= 0 && yy < Dy && xx >= 0 && xx < Dx && !(j == 0 && k == 0) && j * j + k * k <= r * r;
          kq[(j + 2) * 5 + k + 2] = in ? M[yy * Dx + xx] : 0ull;
        }
#pragma unroll
      for (int j = -2; j <= 2; ++j)
#pragma unroll
        for (int k = -2; k <= 2; ++k) {
          const unsigned long long v = kq[(j + 2) * 5 + k + 2];
          const unsigned sq = (unsigned)(v >> 32);
          if (v && (sq > si || (sq == si && (y + j) * Dx + x + k < d.pix))) keep = false;
        }
    } else {
      for (int j = -r; j <= r && keep; ++j) {
        const int yy = y + j;
        if (yy < 0 || yy >= Dy) continue;
        for (int k = -r; k <= r; ++k) {
          const int xx = x + k;
          if (xx < 0 || xx >= Dx || (j == 0 && k == 0) || j * j + k * k > r * r) continue;
          const int q = yy * Dx + xx;
          const unsigned long long kq = M[q];
          if (!kq) continue;
          const unsigned sq = (unsigned)(kq >> 32);
          if (sq > si || (sq == si && q < d.pix)) { keep = false; break; }
        }
      }
    }
    if (keep) {
      const int o = atomicAdd(tmp_n, 1);
      tmp_pos[o] = d.pix; tmp_plane[o] = d.plane; tmp_snr[o] = d.snr;
    }
  }
}

// rank sort by pixel (pixels are distinct) + reset of the touched map entries
__global__ void __launch_bounds__(CAT_THREADS)
k_dedupe_sort(const lpf_det* __restrict__ dets, const int32_t* __restrict__ ndets, int max_det,
              unsigned long long* __restrict__ M, const int32_t* __restrict__ tmp_pos,
              const int16_t* __restrict__ tmp_plane, const float* __restrict__ tmp_snr,
              const int32_t* __restrict__ tmp_n, int32_t* __restrict__ upos, int16_t* __restrict__ uplane,
              float* __restrict__ usnr, int32_t* __restrict__ nu) {
  __shared__ int s_pos[SORT_CAP];
  const int n = min(*ndets, max_det);
  const int m = *tmp_n;
  const bool staged = m <= SORT_CAP;
  if (staged) {
    for (int j = threadIdx.x; j < m; j += blockDim.x) s_pos[j] = tmp_pos[j];
    for (int j = m + threadIdx.x; j < ((m + 3) & ~3); j += blockDim.x) s_pos[j] = 0x7fffffff;
    __syncthreads();
  }
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < m; i += gridDim.x * blockDim.x) {
    const int mine = tmp_pos[i];
    int rank = 0;
    if (staged) {
      const int4* p4 = reinterpret_cast<const int4*>(s_pos);
      for (int j = 0; j < (m + 3) / 4; ++j) {
        const int4 v = p4[j];
        rank += (v.x < mine) + (v.y < mine) + (v.z < mine) + (v.w < mine);
      }
    } else {
      for (int j = 0; j < m; ++j) rank += (tmp_pos[j] < mine);
    }
    upos[rank] = mine; uplane[rank] = tmp_plane[i]; usnr[rank] = tmp_snr[i];
  }
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) M[dets[i].pix] = 0ull;
  if (blockIdx.x == 0 && threadIdx.x == 0) *nu = m;
}

// ---------------------------------------------------------------------------------------------
// nearest active candidate of every unique detection (thread i0, i0 + stride, ...)
__device__ __forceinline__ void
assoc_match_body(const int32_t* __restrict__ upos, const int32_t* __restrict__ nu, const uint8_t* __restrict__ band_ok,
                 int B, const int32_t* __restrict__ slotmap, const int32_t* __restrict__ cpix, int Dy, int Dx, int r,
                 long long t, long long* __restrict__ matched_t, int32_t* __restrict__ cand_idx, int i0, int stride) {
  (void)cpix;
  const int n = *nu;
  const bool frame_ok = band_ok[B] != 0;
  for (int i = i0; i < n; i += stride) {
    int best = -1;
    if (frame_ok) {
      const int pix = upos[i];
      const int y = pix / Dx, x = pix - y * Dx;
      int best_d = 0x7fffffff;
      if (r <= 3) {
        int sl[49];
#pragma unroll
        for (int j = -3; j <= 3; ++j)
#pragma unroll
          for (int k = -3; k <= 3; ++k) {
            const int yy = y + j, xx = x + k;
            const bool in = yy >= 0 && yy < Dy && xx >= 0 && xx < Dx && j * j + k * k <= r * r;
            sl[(j + 3) * 7 + k + 3] = in ? slotmap[yy * Dx + xx] : -1;
          }
#pragma unroll
        for (int j = -3; j <= 3; ++j)
#pragma unroll
          for (int k = -3; k <= 3; ++k) {
            const int s = sl[(j + 3) * 7 + k + 3], d2 = j * j + k * k;
            if (s >= 0 && (d2 < best_d || (d2 == best_d && s < best))) { best_d = d2; best = s; }
          }
      } else
      for (int j = -r; j <= r; ++j) {
        const int yy = y + j;
        if (yy < 0 || yy >= Dy) continue;
        for (int k = -r; k <= r; ++k) {
          const int xx = x + k;
          const int d2 = j * j + k * k;
          if (xx < 0 || xx >= Dx || d2 > r * r) continue;
          const int s = slotmap[yy * Dx + xx];
          if (s < 0) continue;
          if (d2 < best_d || (d2 == best_d && s < best)) { best_d = d2; best = s; }
        }
      }
      if (best >= 0) matched_t[best] = t;
    }
    cand_idx[i] = best;
  }
}

// exclusive block scan of one int per thread (1024 threads)
__device__ __forceinline__ int block_excl_scan(int v, int* s_warp /*[33]*/, int& total) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  int inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const int u = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += u; }
  __syncthreads();
  if (lane == 31) s_warp[w] = inc;
  __syncthreads();
  if (w == 0) {
    int x = lane < (int)(blockDim.x >> 5) ? s_warp[lane] : 0;
    int xi = x;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const int u = __shfl_up_sync(0xffffffffu, xi, o); if (lane >= o) xi += u; }
    s_warp[lane] = xi - x;
    if (lane == 31) s_warp[32] = xi;
  }
  __syncthreads();
  total = s_warp[32];
  return s_warp[w] + inc - v;
}

struct AssocArgs {
  uint8_t* active; uint8_t* forced; int32_t* cpix; int32_t* miss; long long* born; const long long* matched_t;
  int32_t* slotmap; int32_t* free_list; int n_cand_max, n_forget;
  const int32_t* upos; const int32_t* nu; const uint8_t* band_ok; int B; long long t;
  int32_t* cand_idx; int32_t* act_slots; int32_t* act_pix; int32_t* npos; int32_t* counters;
};

// Single block: age / retire, rebuild the slot map around retired pixels, hand the lowest free
// slots to the unmatched detections in ascending pix, compact the active list.  A warp owns a run of
// consecutive slots and walks it 32 at a time (lane = slot: every table access is coalesced); ordered
// compaction by ballot + popc within a step, a running offset across steps, a scan of the warp totals across
// warps.
__device__ __forceinline__ int warp_totals_excl(int my_total, int* s_tot /*[33]*/, int& grand) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
  __syncthreads();
  if (lane == 0) s_tot[w] = my_total;
  __syncthreads();
  int pre = 0, all = 0;
  for (int i = 0; i < nw; ++i) { const int v = s_tot[i]; all += v; if (i < w) pre += v; }
  grand = all;
  return pre;
}

__device__ __forceinline__ void assoc_update_body(const AssocArgs& a) {
  __shared__ int s_warp[33];
  const int T = blockDim.x;
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5, nw = T >> 5;
  const unsigned lt = (1u << lane) - 1u;
  const bool frame_ok = a.band_ok[a.B] != 0;
  // Slots are handed out lowest first, so the table is dense at the bottom: counters[4] is one more than the highest
  // slot ever used, everything from there on is free, and the passes below walk only the slots before it (rounded
  // up to 32) - on the one serial chain of the path this is what the step costs.
  const int hwm0 = __ldcg(&a.counters[4]);
  const int n_scan = min(a.n_cand_max, (hwm0 + 31) & ~31);
  int spw = ((n_scan + nw - 1) / nw + 31) & ~31;          // slots per warp, a multiple of 32
  int w0 = min(w * spw, n_scan), w1 = min(w0 + spw, n_scan);
  if (frame_ok) {
    // 1. age and retire
    int any_retired = 0;
#pragma unroll 4
    for (int s = w0 + lane; s < w1; s += 32) {
      const uint8_t act = a.active[s], frc = a.forced[s];      // independent loads: they leave together
      const long long mt = a.matched_t[s];
      const int m0 = a.miss[s], px = a.cpix[s];
      if (!act) continue;
      const bool hit = mt == a.t;
      const int m = hit ? 0 : m0 + 1;
      if (m != m0) a.miss[s] = m;
      if (!hit && !frc && m >= a.n_forget) { a.active[s] = 0; a.slotmap[px] = -1; any_retired = 1; }
    }
    // 2. another (forced) candidate may share a retired pixel: restore the lowest active slot there
    if (__syncthreads_or(any_retired)) {
      for (int s = w0 + lane; s < w1; s += 32)
        if (a.active[s]) atomicMin(reinterpret_cast<unsigned*>(&a.slotmap[a.cpix[s]]), (unsigned)s);
    }
    // 3. free list (ascending)
    int nfree_w = 0;
    for (int s0 = w0; s0 < w1; s0 += 32) {
      const int s = s0 + lane;
      nfree_w += __popc(__ballot_sync(0xffffffffu, s < w1 && !a.active[s]));
    }
    int n_free_low;
    int off = warp_totals_excl(nfree_w, s_warp, n_free_low);
    const int n_free = n_free_low + (a.n_cand_max - n_scan);      // every slot from n_scan on is free
    for (int s0 = w0; s0 < w1; s0 += 32) {
      const int s = s0 + lane;
      const bool fr = s < w1 && !a.active[s];
      const unsigned m = __ballot_sync(0xffffffffu, fr);
      if (fr) a.free_list[off + __popc(m & lt)] = s;
      off += __popc(m);
    }
    __syncthreads();
    // 4. unmatched detections, ascending pix (upos is sorted)
    const int nu = *a.nu;
    const int peru = (nu + T - 1) / T;
    const int u0 = min(tid * peru, nu), u1 = min(u0 + peru, nu);
    int nun_mine = 0;
    for (int i = u0; i < u1; ++i) nun_mine += (a.cand_idx[i] < 0);
    int n_un;
    int uo = block_excl_scan(nun_mine, s_warp, n_un);
    for (int i = u0; i < u1; ++i) {
      if (a.cand_idx[i] >= 0) continue;
      const int k = uo++;
      if (k < n_free) {
        const int s = k < n_free_low ? a.free_list[k] : n_scan + (k - n_free_low);
        const int pix = a.upos[i];
        if (s >= hwm0) atomicMax(&a.counters[4], s + 1);
        a.active[s] = 1; a.forced[s] = 0; a.cpix[s] = pix; a.miss[s] = 0; a.born[s] = a.t;
        atomicMin(reinterpret_cast<unsigned*>(&a.slotmap[pix]), (unsigned)s);
        a.cand_idx[i] = s;
      } else {
        atomicAdd(&a.counters[1], 1);
      }
    }
    __syncthreads();
  }
  // 5. active list, ascending slot (the slots handed out above may lie beyond n_scan: walk up to the new mark)
  {
    const int n_scan1 = min(a.n_cand_max, (__ldcg(&a.counters[4]) + 31) & ~31);      // (after phase 4's block barrier; past L1)
    spw = ((n_scan1 + nw - 1) / nw + 31) & ~31;
    w0 = min(w * spw, n_scan1); w1 = min(w0 + spw, n_scan1);
  }
  int nact_w = 0;
  for (int s0 = w0; s0 < w1; s0 += 32) {
    const int s = s0 + lane;
    nact_w += __popc(__ballot_sync(0xffffffffu, s < w1 && a.active[s]));
  }
  int n_act;
  int ao = warp_totals_excl(nact_w, s_warp, n_act);
  for (int s0 = w0; s0 < w1; s0 += 32) {
    const int s = s0 + lane;
    const bool ac = s < w1 && a.active[s];
    const int px = s < w1 ? a.cpix[s] : 0;
    const unsigned m = __ballot_sync(0xffffffffu, ac);
    if (ac) { const int o = ao + __popc(m & lt); a.act_slots[o] = s; a.act_pix[o] = px; }
    ao += __popc(m);
  }
  if (tid == 0) { *a.npos = n_act; a.counters[2] = n_act; }
}

// S10 in one block: match (every thread takes detections), then the table update.  One launch, no second
// trip through the block scheduler on the part of a frame that the next frame has to wait for.
__global__ void __launch_bounds__(1024)
k_assoc(const AssocArgs a, int Dy, int Dx, int r, long long* matched_t) {
  assoc_match_body(a.upos, a.nu, a.band_ok, a.B, a.slotmap, a.cpix, Dy, Dx, r, a.t, matched_t, a.cand_idx, threadIdx.x, blockDim.x);
  __syncthreads();       // matched_t and cand_idx (global) are this block's own writes
  assoc_update_body(a);
}

struct AddArgs {
  uint8_t* active; uint8_t* forced; int32_t* cpix; int32_t* miss; long long* born; int32_t* slotmap;
  int32_t* free_list; int n_cand_max; const int32_t* pix; int n; int32_t* slots_out; int32_t* status;
  int n_pix;        // pixels of the image: a position outside [0, n_pix) refuses the whole call (status 2)
  int32_t* n_active; // the context's count of active candidates
  int32_t* hwm;      // one more than the highest slot ever used (k_assoc walks only the slots before it)
};

__global__ void __launch_bounds__(1024)
k_add_candidates(const AddArgs a) {
  __shared__ int s_warp[33];
  const int T = blockDim.x, tid = threadIdx.x;
  const int per = (a.n_cand_max + T - 1) / T;
  const int s0 = tid * per, s1 = min(s0 + per, a.n_cand_max);
  int nfree_mine = 0;
  for (int s = s0; s < s1; ++s) nfree_mine += a.active[s] ? 0 : 1;
  int n_free;
  int off = block_excl_scan(nfree_mine, s_warp, n_free);
  for (int s = s0; s < s1; ++s) if (!a.active[s]) a.free_list[off++] = s;
  __syncthreads();
  if (n_free < a.n) { if (tid == 0) *a.status = 1; return; }
  int bad = 0;
  for (int i = tid; i < a.n; i += T) bad |= (a.pix[i] < 0 || a.pix[i] >= a.n_pix) ? 1 : 0;
  if (__syncthreads_or(bad)) { if (tid == 0) *a.status = 2; return; }
  for (int i = tid; i < a.n; i += T) {
    const int s = a.free_list[i];
    a.active[s] = 1; a.forced[s] = 1; a.cpix[s] = a.pix[i]; a.miss[s] = 0; a.born[s] = -1;
    atomicMin(reinterpret_cast<unsigned*>(&a.slotmap[a.pix[i]]), (unsigned)s);
    atomicMax(a.hwm, s + 1);
    if (a.slots_out) a.slots_out[i] = s;
  }
  if (tid == 0) { *a.status = 0; *a.n_active += a.n; }
}

// NaN rows for freshly added forced slots (slots_out list)
__global__ void __launch_bounds__(256)
k_ring_nan_slots(float* __restrict__ ring, const int32_t* __restrict__ free_list, int n, long long per_slot) {
  for (int i = blockIdx.y; i < n; i += gridDim.y) {
    float* r = ring + (long long)free_list[i] * per_slot;
    for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < per_slot; q += (long long)gridDim.x * blockDim.x)
      r[q] = CUDART_NAN_F;
  }
}

// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_measure_flux(const LpfFrameDesc* __restrict__ fd, const float* __restrict__ cube_arg, const uint8_t* __restrict__ band_ok,
               const uint8_t* __restrict__ W, int B, int Dy, int Dx, int r, const int32_t* __restrict__ pos,
               const int32_t* __restrict__ npos, float* __restrict__ flux) {
  const float* __restrict__ cube = fd ? fd->cube : cube_arg;
  const long long N = (long long)Dy * Dx;
  const long long total = (long long)(*npos) * B;
  const bool frame_ok = band_ok[B] != 0;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
    const int ip = (int)(i / B), b = (int)(i - (long long)ip * B);
    float best = 0.f;
    if (frame_ok && band_ok[b]) {
      const int pix = pos[ip];
      const int y = pix / Dx, x = pix - y * Dx;
      const float* X = cube + (long long)b * N;
      bool any = false;
      for (int j = -r; j <= r; ++j) {
        const int yy = y + j;
        if (yy < 0 || yy >= Dy) continue;
        for (int k = -r; k <= r; ++k) {
          const int xx = x + k;
          if (xx < 0 || xx >= Dx) continue;
          const long long q = (long long)yy * Dx + xx;
          if (!W[q]) continue;
          const float v = __ldg(X + q);
          if (!any || v > best) { best = v; any = true; }
        }
      }
      if (!any) best = 0.f;
    }
    flux[i] = best;
  }
}

// one warp per position: NaN prefill of a slot born at t, then this step's column
__global__ void __launch_bounds__(256)
k_append(float* __restrict__ ring, long long* __restrict__ meta_t, unsigned long long* __restrict__ meta_ok,
         const long long* __restrict__ born, int T_ring, int B, const int32_t* __restrict__ slots,
         const int32_t* __restrict__ n, const float* __restrict__ flux, const uint8_t* __restrict__ band_ok, long long t_arg,
         const LpfFrameDesc* __restrict__ fd) {
  const long long t = fd ? fd->t : t_arg;
  const int tau = (int)(t % T_ring);
  const int lane = threadIdx.x & 31;
  const int wid = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nw = (gridDim.x * blockDim.x) >> 5;
  const int cnt = *n;
  for (int i = wid; i < cnt; i += nw) {
    const int s = slots[i];
    float* r = ring + (long long)s * T_ring * B;
    if (born[s] == t) {
      for (int q = lane; q < T_ring * B; q += 32) r[q] = CUDART_NAN_F;
      __syncwarp();
    }
    for (int b = lane; b < B; b += 32) r[(long long)tau * B + b] = flux[(long long)i * B + b];
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    meta_t[tau] = t;
    unsigned long long bits = 0;
    if (band_ok[B]) for (int b = 0; b < B; ++b) if (band_ok[b]) bits |= (1ull << b);
    meta_ok[tau] = bits;
  }
}

// O11, backward fill: one warp per active position; a slot born at t gets, for every cached
// frame tau in [t - n_back, t - 1] whose ring column still belongs to tau, the O9 flux of that frame at its
// pixel.  Thread 0 of the grid then labels the cache entry that the caller overwrites with frame t next.
struct BackfillArgs {
  float* ring; const long long* meta_t; const long long* born; int T_ring, B, Dy, Dx, r, n_back, depth;
  const int32_t* slots; const int32_t* pix; const int32_t* n;
  const float* cache; const uint8_t* cache_ok; long long* cache_t; const uint8_t* W; long long t;
};

__global__ void __launch_bounds__(256)
k_backfill(const BackfillArgs a) {
  const int lane = threadIdx.x & 31;
  const int wid = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nw = (gridDim.x * blockDim.x) >> 5;
  const int cnt = *a.n;
  const long long N = (long long)a.Dy * a.Dx;
  // one warp per (active position, cache entry): the few new slots' loads do not queue up behind each other
  for (long long job = wid; job < (long long)cnt * a.depth; job += nw) {
    const int i = (int)(job / a.depth), e = (int)(job - (long long)i * a.depth);
    const int s = a.slots[i];
    const long long tau = a.cache_t[e];
    const int pix = a.pix[i];
    if (a.born[s] != a.t) continue;
    const int y = pix / a.Dx, x = pix - y * a.Dx;
    {
      if (tau < 0 || tau < a.t - a.n_back || tau >= a.t) continue;
      const int col = (int)(tau % a.T_ring);
      if (a.meta_t[col] != tau) continue;                 // the ring has moved on: that column is a newer frame's
      const uint8_t* ok = a.cache_ok + (long long)e * (a.B + 1);
      const bool frame_ok = ok[a.B] != 0;
      for (int b = lane; b < a.B; b += 32) {
        float best = 0.f;
        if (frame_ok && ok[b]) {
          const float* X = a.cache + ((long long)e * a.B + b) * N;
          bool any = false;
          for (int j = -a.r; j <= a.r; ++j) {
            const int yy = y + j;
            if (yy < 0 || yy >= a.Dy) continue;
            for (int k = -a.r; k <= a.r; ++k) {
              const int xx = x + k;
              if (xx < 0 || xx >= a.Dx) continue;
              const long long q = (long long)yy * a.Dx + xx;
              if (!a.W[q]) continue;
              const float v = __ldg(X + q);
              if (!any || v > best) { best = v; any = true; }
            }
          }
          if (!any) best = 0.f;
        }
        a.ring[((long long)s * a.T_ring + col) * a.B + b] = best;
      }
    }
  }
}

// labels cache entry e with frame t (after the copies that fill it were enqueued)
__global__ void k_cache_label(long long* cache_t, int e, long long t) { cache_t[e] = t; }

__global__ void __launch_bounds__(256)
k_get_dynspec(const float* __restrict__ ring, const long long* __restrict__ meta_t, int T_ring, int B, int slot,
              long long t_last, float* __restrict__ out) {
  const float* r = ring + (long long)slot * T_ring * B;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < B * T_ring; i += gridDim.x * blockDim.x) {
    const int b = i / T_ring, j = i - b * T_ring;
    const long long tt = t_last - T_ring + 1 + j;
    const int tau = (int)(((tt % T_ring) + T_ring) % T_ring);
    const bool have = tt >= 0 && meta_t[tau] == tt;
    out[i] = have ? r[(long long)tau * B + b] : CUDART_NAN_F;
  }
}

__global__ void k_fill_f32(float* p, long long n, float v) {
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) p[i] = v;
}
__global__ void k_fill_i32(int32_t* p, long long n, int32_t v) {
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) p[i] = v;
}

}  // namespace

int lpf_launch_dedupe(lpf_ctx* c, LpfLane& L, const lpf_det* d_dets, const int32_t* d_ndets, int32_t* d_upos,
                      int16_t* d_uplane, float* d_usnr, int32_t* d_nu, cudaStream_t st) {
  const lpf_params& p = c->p;
  LPF_KLAUNCH(c, KID_DEDUPE_SCATTER, st, k_dedupe_scatter<<<CAT_BLOCKS, CAT_THREADS, 0, st>>>(
      d_dets, d_ndets, p.max_det, L.M, L.tmp_n));
  LPF_KLAUNCH(c, KID_DEDUPE_SELECT, st, k_dedupe_select<<<CAT_BLOCKS, CAT_THREADS, 0, st>>>(
      d_dets, d_ndets, p.max_det, L.M, p.Dy, p.Dx, p.r_dedupe, L.tmp_pos, L.tmp_plane, L.tmp_snr, L.tmp_n));
  LPF_KLAUNCH(c, KID_DEDUPE_SORT, st, k_dedupe_sort<<<CAT_BLOCKS, CAT_THREADS, 0, st>>>(
      d_dets, d_ndets, p.max_det, L.M, L.tmp_pos, L.tmp_plane, L.tmp_snr, L.tmp_n, d_upos, d_uplane, d_usnr, d_nu));
  return LPF_OK;
}

int lpf_launch_associate(lpf_ctx* c, const int32_t* d_upos, const int32_t* d_nu, const uint8_t* d_band_ok,
                         long long t, int32_t* d_cand_idx, int32_t* d_act_slots, int32_t* d_act_pix,
                         int32_t* d_npos, cudaStream_t st) {
  const lpf_params& p = c->p;
  AssocArgs a{};
  a.active = c->active; a.forced = c->forced; a.cpix = c->cpix; a.miss = c->miss; a.born = c->born;
  a.matched_t = c->matched_t; a.slotmap = c->slotmap; a.free_list = c->free_list;
  a.n_cand_max = p.n_cand_max; a.n_forget = p.n_forget;
  a.upos = d_upos; a.nu = d_nu; a.band_ok = d_band_ok; a.B = p.B; a.t = t;
  a.cand_idx = d_cand_idx; a.act_slots = d_act_slots; a.act_pix = d_act_pix; a.npos = d_npos; a.counters = c->counters;
  LPF_KLAUNCH(c, KID_ASSOC_UPDATE, st, k_assoc<<<1, 1024, 0, st>>>(a, p.Dy, p.Dx, p.r_assoc, c->matched_t));
  return LPF_OK;
}

int lpf_launch_add_candidates(lpf_ctx* c, const int32_t* d_pix, int n, int32_t* d_slots_out, cudaStream_t st) {
  const lpf_params& p = c->p;
  int32_t* d_status = c->counters + 3;
  AddArgs a{};
  a.active = c->active; a.forced = c->forced; a.cpix = c->cpix; a.miss = c->miss; a.born = c->born;
  a.slotmap = c->slotmap; a.free_list = c->free_list; a.n_cand_max = p.n_cand_max;
  a.pix = d_pix; a.n = n; a.slots_out = d_slots_out; a.status = d_status; a.n_pix = (int)c->N; a.n_active = c->counters + 2; a.hwm = c->counters + 4;
  LPF_KLAUNCH(c, KID_MISC, st, k_add_candidates<<<1, 1024, 0, st>>>(a));
  int32_t status = -1;
  LPF_CUDA(cudaMemcpyAsync(&status, d_status, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
  LPF_CUDA(cudaStreamSynchronize(st));
  if (status == 2) return LPF_E_ARG;
  if (status != 0) return LPF_E_STATE;
  if (n > 0) {
    const long long per_slot = (long long)p.T_ring * p.B;
    const long long gx = (per_slot + 255) / 256;
    const dim3 grid((unsigned)(gx < 64 ? gx : 64), (unsigned)(n < 4096 ? n : 4096));
    LPF_KLAUNCH(c, KID_MISC, st, k_ring_nan_slots<<<grid, 256, 0, st>>>(c->ring, c->free_list, n, per_slot));
    LPF_CUDA(cudaStreamSynchronize(st));
  }
  return LPF_OK;
}

int lpf_launch_measure_flux(lpf_ctx* c, const float* d_cube, const uint8_t* d_band_ok, const int32_t* d_pos,
                            const int32_t* d_npos, float* d_flux, cudaStream_t st) {
  const lpf_params& p = c->p;
  LPF_KLAUNCH(c, KID_MEASURE_FLUX, st, k_measure_flux<<<c->n_sm * 2, 256, 0, st>>>(
      c->cap_fd, d_cube, d_band_ok, c->W, p.B, p.Dy, p.Dx, p.r_flux, d_pos, d_npos, d_flux));
  return LPF_OK;
}

int lpf_launch_append(lpf_ctx* c, const int32_t* d_slots, const int32_t* d_n, const float* d_flux,
                      const uint8_t* d_band_ok, long long t, cudaStream_t st) {
  const lpf_params& p = c->p;
  LPF_KLAUNCH(c, KID_APPEND, st, k_append<<<c->n_sm, 256, 0, st>>>(
      c->ring, c->meta_t, c->meta_ok, c->born, p.T_ring, p.B, d_slots, d_n, d_flux, d_band_ok, t, c->cap_fd));
  return LPF_OK;
}

int lpf_launch_backfill(lpf_ctx* c, const int32_t* d_slots, const int32_t* d_pix, const int32_t* d_n, const float* d_cube,
                        const uint8_t* d_band_ok, long long t, cudaStream_t st) {
  const lpf_params& p = c->p;
  BackfillArgs a{};
  a.ring = c->ring; a.meta_t = c->meta_t; a.born = c->born; a.T_ring = p.T_ring; a.B = p.B; a.Dy = p.Dy; a.Dx = p.Dx;
  a.r = p.r_flux; a.n_back = p.n_back; a.depth = p.n_back + p.n_lanes; a.slots = d_slots; a.pix = d_pix; a.n = d_n;
  a.cache = c->cube_cache; a.cache_ok = c->cache_ok; a.cache_t = c->cache_t; a.W = c->W; a.t = t;
  LPF_KLAUNCH(c, KID_BACKFILL, st, k_backfill<<<c->n_sm * 2, 256, 0, st>>>(a));
  return LPF_OK;
}

// Frame t joins the cache.  The cache holds n_back + n_lanes entries, so the entry that frame t overwrites
// (frame t - n_back - n_lanes) is older than anything a frame still in flight on another lane back-fills from:
// the copy needs no ordering against the other lanes and overlaps the lane's own detection kernel.
int lpf_launch_cache_store(lpf_ctx* c, const float* d_cube, const uint8_t* d_band_ok, long long t, cudaStream_t st) {
  const lpf_params& p = c->p;
  const int e = (int)(t % (p.n_back + p.n_lanes));
  const size_t cube_elems = (size_t)p.B * c->N;
  LPF_CUDA(cudaMemcpyAsync(c->cube_cache + (size_t)e * cube_elems, d_cube, cube_elems * sizeof(float), cudaMemcpyDeviceToDevice, st));
  LPF_CUDA(cudaMemcpyAsync(c->cache_ok + (size_t)e * (p.B + 1), d_band_ok, (size_t)p.B + 1, cudaMemcpyDeviceToDevice, st));
  LPF_KLAUNCH(c, KID_MISC, st, k_cache_label<<<1, 1, 0, st>>>(c->cache_t, e, t));
  return LPF_OK;
}

// O13: [n][B][T_ring] time-ordered, sigma-normalised, NaN-free dynamic spectra of a list of slots
__global__ void __launch_bounds__(256)
k_export_dynspec(const float* __restrict__ ring, const long long* __restrict__ meta_t, int T_ring, int B, int n_cand_max,
                 const int32_t* __restrict__ slots, int n, long long t_last, const float* __restrict__ sigma, float* __restrict__ out) {
  const long long per = (long long)B * T_ring, total = per * n;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
    const int is = (int)(i / per);
    const int r = (int)(i - (long long)is * per);
    const int b = r / T_ring, j = r - b * T_ring;
    const int slot = slots[is];
    float v = 0.f;
    if (slot >= 0 && slot < n_cand_max) {
      const long long tt = t_last - T_ring + 1 + j;
      const int tau = (int)(((tt % T_ring) + T_ring) % T_ring);
      if (tt >= 0 && meta_t[tau] == tt) {
        const float x = ring[((long long)slot * T_ring + tau) * B + b];
        const float sg = sigma ? sigma[b] : 1.f;
        if (x == x) v = (float)((double)x / (double)(sg > 0.f ? sg : 1.f));
      }
    }
    out[i] = v;
  }
}

// O14: eqs. 19-21, one thread per (sample, band, time step)
__global__ void __launch_bounds__(256)
k_simulate_pulses(int n, int B, int T, const float* __restrict__ nu, float nu0, float dt_s, const float* __restrict__ theta,
                  float* __restrict__ out, int accumulate) {
  const long long per = (long long)B * T, total = per * n;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
    const int is = (int)(i / per);
    const int r = (int)(i - (long long)is * per);
    const int b = r / T, j = r - b * T;
    const float* th = theta + 5 * is;
    const float t0 = th[0], w = th[1], dm = th[2], A = th[3], al = th[4];
    const float v = nu[b];
    const float tn = t0 + 4148.806f * dm * (1.f / (v * v) - 1.f / (nu0 * nu0)) / dt_s;      // eq. 20
    const float u = ((float)j - tn) / w;
    const float I = A * powf(v / nu0, al) * expf(-0.5f * u * u);                              // eqs. 19, 21
    out[i] = accumulate ? out[i] + I : I;
  }
}

int lpf_launch_export_dynspec(lpf_ctx* c, const int32_t* d_slots, int n, long long t_last, const float* d_sigma, float* d_out,
                              cudaStream_t st) {
  const lpf_params& p = c->p;
  const long long total = (long long)n * p.B * p.T_ring;
  const int blocks = (int)std::min<long long>((total + 255) / 256, (long long)c->n_sm * 8);
  LPF_KLAUNCH(c, KID_MISC, st, k_export_dynspec<<<blocks, 256, 0, st>>>(c->ring, c->meta_t, p.T_ring, p.B, p.n_cand_max, d_slots, n,
                                                                       t_last, d_sigma, d_out));
  return LPF_OK;
}

int lpf_launch_simulate_pulses(int n, int B, int T, const float* d_nu, float nu0, float dt_s, const float* d_theta, float* d_out,
                               int accumulate, cudaStream_t st) {
  const long long total = (long long)n * B * T;
  int dev = 0, n_sm = 148;
  if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
  const int blocks = (int)std::min<long long>((total + 255) / 256, (long long)n_sm * 16);
  k_simulate_pulses<<<blocks, 256, 0, st>>>(n, B, T, d_nu, nu0, dt_s, d_theta, d_out, accumulate);
  cudaError_t e = cudaPeekAtLastError();
  if (e != cudaSuccess) return lpf_cuda_fail(e, "k_simulate_pulses");
  return LPF_OK;
}

int lpf_launch_get_dynspec(lpf_ctx* c, int slot, long long t_last, float* d_out, cudaStream_t st) {
  const lpf_params& p = c->p;
  LPF_KLAUNCH(c, KID_MISC, st, k_get_dynspec<<<8, 256, 0, st>>>(c->ring, c->meta_t, p.T_ring, p.B, slot, t_last, d_out));
  return LPF_OK;
}

int lpf_launch_fill_nan(lpf_ctx* c, float* d, int64_t n, cudaStream_t st) {
  LPF_KLAUNCH(c, KID_MISC, st, k_fill_f32<<<c->n_sm * 4, 256, 0, st>>>(d, n, nanf("")));
  return LPF_OK;
}
int lpf_launch_fill_i32(lpf_ctx* c, int32_t* d, int64_t n, int32_t v, cudaStream_t st) {
  LPF_KLAUNCH(c, KID_MISC, st, k_fill_i32<<<c->n_sm * 4, 256, 0, st>>>(d, n, v));
  return LPF_OK;
}
