// C-ABI entry points (include/lpf.h): argument checks, context life cycle, step chaining.
#include <algorithm>
#include <climits>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>

#include "lpf_internal.cuh"

thread_local char g_lpf_cuda_err[256] = "";

int lpf_cuda_fail(cudaError_t e, const char* what) {
  snprintf(g_lpf_cuda_err, sizeof(g_lpf_cuda_err), "%s: %s", what, cudaGetErrorString(e));
  (void)cudaGetLastError();
  return LPF_E_CUDA;
}

static cudaEvent_t prof_event(lpf_ctx* c) {
  if (c->prof_pool_used == c->prof_pool.size()) {
    cudaEvent_t e = nullptr;
    cudaEventCreate(&e);
    c->prof_pool.push_back(e);
  }
  return c->prof_pool[c->prof_pool_used++];
}

void lpf_prof_pre(lpf_ctx* c, int kid, cudaStream_t st) {
  lpf_ctx::ProfRec r;
  r.kid = kid; r.e0 = prof_event(c); r.e1 = prof_event(c);
  cudaEventRecord(r.e0, st);
  c->prof_recs.push_back(r);
}

void lpf_prof_post(lpf_ctx* c, cudaStream_t st) { cudaEventRecord(c->prof_recs.back().e1, st); }

namespace {

// eq. 2 taps, R1: g_i = exp(-i^2 / 2 s^2) / sum ; uniform: 1/(2k+1) ; s <= 0: identity.
void make_taps(int kind, double s, int k, LpfTaps* t) {
  t->R = k;
  const int n = 2 * k + 1;
  double e[LPF_NTAPS];
  double sum = 0;
  for (int i = -k; i <= k; ++i) {
    double v;
    if (kind == 1) v = 1.0;
    else if (s <= 0) v = (i == 0) ? 1.0 : 0.0;
    else v = std::exp(-(double)(i * i) / (2.0 * s * s));
    e[i + k] = v; sum += v;
  }
  for (int i = 0; i < LPF_NTAPS; ++i) t->g[i] = i < n ? (float)(e[i] / sum) : 0.f;
}

template <typename T>
int dalloc(T** p, size_t n) {
  cudaError_t e = cudaMalloc((void**)p, n * sizeof(T));
  if (e != cudaSuccess) { lpf_cuda_fail(e, "cudaMalloc"); return LPF_E_NOMEM; }
  return LPF_OK;
}

#define TRY(x) do { int rc__ = (x); if (rc__ != LPF_OK) return rc__; } while (0)

int check_params(const lpf_params* p) {
  if (!p) return LPF_E_ARG;
  if (p->B < 1 || p->B > LPF_MAX_BANDS || p->Dy < 1 || p->Dx < 1) return LPF_E_ARG;
  if ((long long)p->Dy * p->Dx > (1ll << 30)) return LPF_E_ARG;
  if (!(p->kappa > 0) || p->k_max < 0 || p->k_max > 8) return LPF_E_ARG;
  if (p->k_mf < 0 || p->k_mf > LPF_MAX_RADIUS || p->k_bg < 1 || p->k_bg > LPF_MAX_RADIUS) return LPF_E_ARG;
  if (p->bg_kernel != 0 && p->bg_kernel != 1) return LPF_E_ARG;
  if (p->force_general != 0 && p->force_general != 1) return LPF_E_ARG;
  if (p->bg_kernel == 0 && !(p->s_bg > 0)) return LPF_E_ARG;
  if (p->n_iter < 1 || p->n_iter > 255) return LPF_E_ARG;
  if (p->r_flux < 0 || p->r_flux > 8 || p->r_dedupe < 0 || p->r_dedupe > 8 || p->r_assoc < 0 || p->r_assoc > 8) return LPF_E_ARG;
  if (p->n_forget < 1 || p->T_ring < 1 || p->n_cand_max < 1 || p->max_det < 1 || p->n_lanes < 1 || p->n_lanes > 64) return LPF_E_ARG;
  if (p->n_back < 0 || p->n_back > 64) return LPF_E_ARG;
  if (!(p->zeta_thr >= 0)) return LPF_E_ARG;
  if (p->zeta_thr > 0 && (p->zeta_nmax < 0 || p->zeta_window < 1 || p->zeta_warm < 2 || p->zeta_reset < 0)) return LPF_E_ARG;
  if (!(p->eps_rel >= 0) || !(p->qc_tau > 0) || !(p->qc_clip > 0)) return LPF_E_ARG;
  return LPF_OK;
}

int alloc_lane(lpf_ctx* c, LpfLane& L) {
  const lpf_params& p = c->p;
  const size_t N = (size_t)c->N;
  TRY(dalloc(&L.qc_part1, (size_t)p.B * std::max(c->qc_nblk, lpf_qs_blocks(c)) * 3));
  TRY(dalloc(&L.qc_part2, (size_t)std::max(lpf_qc2_blocks(c), lpf_qs_blocks(c)) * p.B * 3));
  TRY(dalloc(&L.qc_mom, (size_t)p.B * 3));
  TRY(dalloc(&L.dirty_b, (size_t)p.B));
  LPF_CUDA(cudaMemset(L.dirty_b, 0, (size_t)p.B * sizeof(int32_t)));
  TRY(dalloc(&L.qc_band_clip, (size_t)p.B * 2));
  TRY(dalloc(&L.qc_counter, 2));
  LPF_CUDA(cudaMemset(L.qc_counter, 0, 2 * sizeof(int32_t)));
  TRY(dalloc(&L.sum_plane, N));
  TRY(dalloc(&L.dirty, 1));
  LPF_CUDA(cudaMemset(L.dirty, 0, sizeof(int32_t)));
  if (!c->fused) TRY(lpf_ensure_general_scratch(c, L));   // with the fused path planned: on first use (a misaligned cube)
  TRY(dalloc(&L.M, N));
  LPF_CUDA(cudaMemset(L.M, 0, N * sizeof(unsigned long long)));
  TRY(dalloc(&L.tmp_pos, (size_t)p.max_det));
  TRY(dalloc(&L.tmp_plane, (size_t)p.max_det));
  TRY(dalloc(&L.tmp_snr, (size_t)p.max_det));
  TRY(dalloc(&L.tmp_n, 1));
  TRY(dalloc(&L.stats, (size_t)p.B * LPF_STATS_PER_BAND));
  TRY(dalloc(&L.big_thr, (size_t)p.B + 1));
  if (c->fused) {
    long long hb = 0, ns = 0;
    lpf_fused_hit_sizes(c->fused, c->n_planes, &hb, &ns);
    TRY(dalloc(reinterpret_cast<char**>(&L.hits), (size_t)hb));
    TRY(dalloc(&L.hit_cnt, (size_t)ns));
    LPF_CUDA(cudaMemset(L.hit_cnt, 0, (size_t)ns * sizeof(int32_t)));
  }
  TRY(dalloc(&L.zeta_cnt, (size_t)p.B));
  LPF_CUDA(cudaMemset(L.zeta_cnt, 0, (size_t)p.B * sizeof(int32_t)));
  TRY(dalloc(&L.band_ok, (size_t)p.B + 1));
  TRY(dalloc(&L.dets, (size_t)p.max_det));
  TRY(dalloc(&L.ndets, 1));
  TRY(dalloc(&L.upos, (size_t)p.max_det));
  TRY(dalloc(&L.uplane, (size_t)p.max_det));
  TRY(dalloc(&L.usnr, (size_t)p.max_det));
  TRY(dalloc(&L.nu, 1));
  TRY(dalloc(&L.cand_idx, (size_t)p.max_det));
  TRY(dalloc(&L.act_slots, (size_t)p.n_cand_max));
  TRY(dalloc(&L.act_pix, (size_t)p.n_cand_max));
  TRY(dalloc(&L.npos, 1));
  TRY(dalloc(&L.flux, (size_t)p.n_cand_max * p.B));
  LPF_CUDA(cudaMemset(L.ndets, 0, sizeof(int32_t)));
  LPF_CUDA(cudaMemset(L.nu, 0, sizeof(int32_t)));
  LPF_CUDA(cudaMemset(L.npos, 0, sizeof(int32_t)));
  LPF_CUDA(cudaMallocHost((void**)&L.h_counts, 4 * sizeof(int32_t)));
  TRY(dalloc(&L.fdesc, 1));
  LPF_CUDA(cudaEventCreateWithFlags(&L.ev_pre, cudaEventDisableTiming));
  LPF_CUDA(cudaEventCreateWithFlags(&L.ev_post, cudaEventDisableTiming));
  return LPF_OK;
}

}  // namespace

// F, C, S (+ Y, per-plane normalisers for n_iter > 1) of the general multi-kernel path: 3 (B + 1) N floats per lane
int lpf_ensure_general_scratch(lpf_ctx* c, LpfLane& L) {
  if (L.F) return LPF_OK;
  const lpf_params& p = c->p;
  const size_t N = (size_t)c->N, P = (size_t)p.B + 1;
  TRY(dalloc(&L.F, P * N));
  TRY(dalloc(&L.C, P * N));
  TRY(dalloc(&L.S, P * N));
  if (p.n_iter > 1) { TRY(dalloc(&L.Y, P * N)); TRY(dalloc(&L.normp, P * N)); }
  return LPF_OK;
}

namespace {

void free_lane(LpfLane& L) {
  void* ptrs[] = {L.qc_part1, L.qc_part2, L.qc_band_clip, L.qc_counter, L.sum_plane, L.dirty, L.F, L.C, L.S, L.Y, L.normp, L.M, L.tmp_pos, L.tmp_plane,
                  L.tmp_snr, L.tmp_n, L.stats, L.band_ok, L.dets, L.ndets, L.upos, L.uplane, L.usnr, L.nu,
                  L.cand_idx, L.act_slots, L.act_pix, L.npos, L.flux, L.cube, L.zeta_cnt, L.hits, L.hit_cnt, L.big_thr, L.dirty_b, L.qc_mom};
  for (void* q : ptrs) if (q) cudaFree(q);
  if (L.h_counts) cudaFreeHost(L.h_counts);
  if (L.gx_a) cudaGraphExecDestroy(L.gx_a);
  if (L.gx_b) cudaGraphExecDestroy(L.gx_b);
  if (L.g_a) cudaGraphDestroy(L.g_a);
  if (L.fdesc) cudaFree(L.fdesc);
  if (L.ev_pre) cudaEventDestroy(L.ev_pre);
  if (L.ev_post) cudaEventDestroy(L.ev_post);
  L = LpfLane();
}

}  // namespace

// S3-S8 dispatch: the fused sweep kernel when the parameter set allows it, else the general path.
int lpf_launch_detect(lpf_ctx* c, LpfLane& L, const float* d_cube, const uint8_t* d_band_ok, lpf_det* d_dets,
                      int32_t* d_ndets, bool sum_done, cudaStream_t st) {
  // the fused kernel fetches rows with 16-byte bulk copies: a misaligned cube takes the general path
  if (c->fused && (((uintptr_t)d_cube) & 15) == 0)
    return lpf_launch_detect_fused(c, c->fused, L, d_cube, d_band_ok, d_dets, d_ndets, sum_done, st);
  TRY(lpf_ensure_general_scratch(c, L));
  return lpf_launch_detect_general(c, L, d_cube, d_band_ok, d_dets, d_ndets, sum_done, st);
}

namespace {

// first node of a lane's graph: the one node whose parameters change from launch to launch
__global__ void k_set_frame(LpfFrameDesc* fd, const float* cube, long long t, int seq) {
  fd->cube = cube; fd->t = t; fd->seq = seq; fd->pad = 0;
}

int seq_of(long long t) { return (int)(t % 0x3ffffff0LL) + 1; }

// The frame chain of a lane without its association step (which runs on the context's own stream): graph A =
// set_frame, QC, detection, duplicate filter; graph B = flux, append.  Captured once per lane on the context's
// capture stream; every pointer in it is lane- or context-owned, what changes per frame comes through the descriptor.
int build_lane_graphs(lpf_ctx* c, LpfLane& L, const float* d_cube, long long t) {
  cudaStream_t cs = c->cap_st;
  cudaGraph_t ga = nullptr, gb = nullptr;
  const int64_t launches0 = c->launches;
  c->cap_fd = L.fdesc;
  int rc = LPF_OK;
  cudaError_t e = cudaStreamBeginCapture(cs, cudaStreamCaptureModeThreadLocal);
  if (e == cudaSuccess) {
    k_set_frame<<<1, 1, 0, cs>>>(L.fdesc, d_cube, t, seq_of(t));
    c->launches++;
    rc = lpf_launch_qc_sum(c, L, d_cube, L.stats, L.band_ok, L.ndets, cs);
    if (!rc) rc = lpf_launch_detect(c, L, d_cube, L.band_ok, L.dets, L.ndets, true, cs);
    if (!rc) rc = lpf_launch_dedupe(c, L, L.dets, L.ndets, L.upos, L.uplane, L.usnr, L.nu, cs);
    e = cudaStreamEndCapture(cs, &ga);
  }
  L.g_nodes_a = (int)(c->launches - launches0);
  const int64_t launches1 = c->launches;
  if (e == cudaSuccess && !rc) {
    e = cudaStreamBeginCapture(cs, cudaStreamCaptureModeThreadLocal);
    if (e == cudaSuccess) {
      rc = lpf_launch_measure_flux(c, d_cube, L.band_ok, L.act_pix, L.npos, L.flux, cs);
      if (!rc) rc = lpf_launch_append(c, L.act_slots, L.npos, L.flux, L.band_ok, t, cs);
      e = cudaStreamEndCapture(cs, &gb);
    }
  }
  L.g_nodes_b = (int)(c->launches - launches1);
  c->launches = launches0;          // nothing has been launched yet
  c->cap_fd = nullptr;
  if (e == cudaSuccess && !rc) e = cudaGraphInstantiate(&L.gx_a, ga, 0);
  if (e == cudaSuccess && !rc) e = cudaGraphInstantiate(&L.gx_b, gb, 0);
  if (e == cudaSuccess && !rc) {     // the descriptor node: the only root of graph A
    size_t n = 1;
    cudaGraphNode_t root = nullptr;
    e = cudaGraphGetRootNodes(ga, &root, &n);
    if (e == cudaSuccess && n >= 1) L.gnode_set = root; else if (e == cudaSuccess) e = cudaErrorUnknown;
  }
  if (gb) cudaGraphDestroy(gb);
  if (e != cudaSuccess || rc) {
    (void)cudaGetLastError();
    if (ga) cudaGraphDestroy(ga);
    if (L.gx_a) { cudaGraphExecDestroy(L.gx_a); L.gx_a = nullptr; }
    if (L.gx_b) { cudaGraphExecDestroy(L.gx_b); L.gx_b = nullptr; }
    L.g_failed = true;
    return rc ? rc : LPF_OK;         // the direct path serves the lane
  }
  L.g_a = ga;                        // the descriptor node's handle belongs to this graph: it lives as long as the lane
  return LPF_OK;
}

int lane_ok(lpf_ctx* c, int lane) { return (c && lane >= 0 && lane < (int)c->lanes.size()) ? LPF_OK : LPF_E_ARG; }

}  // namespace

extern "C" {

int lpf_create(lpf_ctx** out, const lpf_params* p, const uint8_t* d_valid_mask) {
  if (!out) return LPF_E_ARG;
  *out = nullptr;
  TRY(check_params(p));
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return lpf_cuda_fail(cudaErrorNoDevice, "cudaGetDeviceCount");
  lpf_ctx* c = new (std::nothrow) lpf_ctx();
  if (!c) return LPF_E_NOMEM;
  c->p = *p;
  c->N = (int64_t)p->Dy * p->Dx;
  c->n_planes = p->B + (p->detect_sum_plane ? 1 : 0);
  {
    long long nb = c->N / 8192;
    c->qc_nblk = (int)(nb < 1 ? 1 : (nb > 64 ? 64 : nb));
  }
  int dev = 0;
  cudaGetDevice(&dev);
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess) { delete c; return lpf_cuda_fail(cudaErrorUnknown, "cudaGetDeviceProperties"); }
  c->n_sm = prop.multiProcessorCount;
  make_taps(0, p->sigma_mf, p->k_mf, &c->g_mf);
  make_taps(p->bg_kernel, p->s_bg, p->k_bg, &c->g_bg);

  auto fail = [&](int rc) { lpf_destroy(c); return rc; };
#define TRYC(x) do { int rc__ = (x); if (rc__ != LPF_OK) return fail(rc__); } while (0)
#define CUDAC(x) do { cudaError_t e__ = (x); if (e__ != cudaSuccess) return fail(lpf_cuda_fail(e__, #x)); } while (0)
  const size_t N = (size_t)c->N;
  TRYC(dalloc(&c->W, N));
  if (d_valid_mask) CUDAC(cudaMemcpy(c->W, d_valid_mask, N, cudaMemcpyDeviceToDevice));
  else CUDAC(cudaMemset(c->W, 1, N));
  {  // first valid pixel: pivot of the band statistics
    std::vector<uint8_t> hW(N);
    CUDAC(cudaMemcpy(hW.data(), c->W, N, cudaMemcpyDeviceToHost));
    c->first_valid = 0;
    for (size_t i = 0; i < N; ++i) if (hW[i]) { c->first_valid = (int)i; break; }
    // normalise to {0,1}
    bool dirty = false;
    for (size_t i = 0; i < N; ++i) if (hW[i] > 1) { hW[i] = 1; dirty = true; }
    if (dirty) CUDAC(cudaMemcpy(c->W, hW.data(), N, cudaMemcpyHostToDevice));
    TRYC(dalloc(&c->norm_mf, N));
    TRYC(dalloc(&c->norm_bg, N));
    TRYC(lpf_general_prepare());
    TRYC(lpf_launch_static_norm(c, c->g_mf, c->norm_mf, nullptr, 0));
    TRYC(lpf_launch_static_norm(c, c->g_bg, c->norm_bg, nullptr, 0));
    TRYC(lpf_fused_plan(c, hW.data(), &c->fused));   // reads norm_mf back for its interior constant
  }

  const size_t nc = (size_t)p->n_cand_max;
  TRYC(dalloc(&c->active, nc)); TRYC(dalloc(&c->forced, nc)); TRYC(dalloc(&c->cpix, nc)); TRYC(dalloc(&c->miss, nc));
  TRYC(dalloc(&c->born, nc)); TRYC(dalloc(&c->matched_t, nc)); TRYC(dalloc(&c->free_list, nc));
  TRYC(dalloc(&c->slotmap, N));
  TRYC(dalloc(&c->ring, nc * p->T_ring * p->B));
  TRYC(dalloc(&c->meta_t, (size_t)p->T_ring)); TRYC(dalloc(&c->meta_ok, (size_t)p->T_ring));
  TRYC(dalloc(&c->counters, 8));
  if (p->zeta_thr > 0) {
    TRYC(dalloc(&c->rq_m, 2 * (size_t)p->B * N));
    TRYC(dalloc(&c->rq_v, 2 * (size_t)p->B * N));
    TRYC(dalloc(&c->rq_state, 4 * (size_t)p->B + 1));
    CUDAC(cudaMemset(c->rq_m, 0, 2 * (size_t)p->B * N * sizeof(float)));
    CUDAC(cudaMemset(c->rq_v, 0, 2 * (size_t)p->B * N * sizeof(float)));
    CUDAC(cudaMemset(c->rq_state, 0, (4 * (size_t)p->B + 1) * sizeof(int32_t)));
    CUDAC(cudaEventCreateWithFlags(&c->rq_ev, cudaEventDisableTiming));
  }
  if (p->n_back > 0) {
    const size_t depth = (size_t)p->n_back + p->n_lanes;
    TRYC(dalloc(&c->cube_cache, depth * p->B * N));
    TRYC(dalloc(&c->cache_ok, depth * (p->B + 1)));
    TRYC(dalloc(&c->cache_t, depth));
    CUDAC(cudaMemset(c->cache_t, 0xff, depth * 8));   // -1
  }
  CUDAC(cudaMemset(c->active, 0, nc)); CUDAC(cudaMemset(c->forced, 0, nc));
  CUDAC(cudaMemset(c->cpix, 0, nc * 4)); CUDAC(cudaMemset(c->miss, 0, nc * 4));
  CUDAC(cudaMemset(c->born, 0xff, nc * 8));       // -1
  CUDAC(cudaMemset(c->matched_t, 0x80, nc * 8));  // very negative
  CUDAC(cudaMemset(c->slotmap, 0xff, N * 4));     // -1
  CUDAC(cudaMemset(c->meta_t, 0xff, (size_t)p->T_ring * 8));
  CUDAC(cudaMemset(c->meta_ok, 0, (size_t)p->T_ring * 8));
  CUDAC(cudaMemset(c->counters, 0, 8 * 4));
  TRYC(lpf_launch_fill_nan(c, c->ring, (int64_t)(nc * p->T_ring * p->B), 0));
  CUDAC(cudaEventCreateWithFlags(&c->ring_ev, cudaEventDisableTiming));
  TRYC(lpf_qc_prepare());
  {
    int lo = 0, hi = 0;
    CUDAC(cudaDeviceGetStreamPriorityRange(&lo, &hi));
    CUDAC(cudaStreamCreateWithPriority(&c->chain_st, cudaStreamNonBlocking, hi));
    CUDAC(cudaStreamCreateWithFlags(&c->cap_st, cudaStreamNonBlocking));
  }
  c->lanes.resize(p->n_lanes);
  for (auto& L : c->lanes) TRYC(alloc_lane(c, L));
  CUDAC(cudaDeviceSynchronize());
  CUDAC(cudaGetLastError());
#undef TRYC
#undef CUDAC
  *out = c;
  return LPF_OK;
}

// ---- checkpoint / resume ------------------------------------------------------------------------------------------
namespace {
struct StateHeader { char magic[8]; int32_t version, params_bytes; int64_t N, total; lpf_params p; };
struct StateSection { void* d; size_t bytes; };

// the device arrays that persist from frame to frame, in the order they are stored
std::vector<StateSection> state_sections(const lpf_ctx* c) {
  const lpf_params& p = c->p;
  const size_t nc = (size_t)p.n_cand_max, N = (size_t)c->N;
  std::vector<StateSection> v = {
      {c->active, nc}, {c->forced, nc}, {c->cpix, nc * 4}, {c->miss, nc * 4}, {c->born, nc * 8}, {c->matched_t, nc * 8},
      {c->slotmap, N * 4}, {c->ring, nc * p.T_ring * p.B * 4}, {c->meta_t, (size_t)p.T_ring * 8}, {c->meta_ok, (size_t)p.T_ring * 8},
      {c->counters, 8 * 4}};
  if (c->rq_m) {
    v.push_back({c->rq_m, 2 * (size_t)p.B * N * 4}); v.push_back({c->rq_v, 2 * (size_t)p.B * N * 4});
    v.push_back({c->rq_state, (4 * (size_t)p.B + 1) * 4});
  }
  if (c->cube_cache) {
    const size_t depth = (size_t)p.n_back + p.n_lanes;
    v.push_back({c->cube_cache, depth * p.B * N * 4}); v.push_back({c->cache_ok, depth * (p.B + 1)});
    v.push_back({c->cache_t, depth * 8});
  }
  return v;
}
}  // namespace

int64_t lpf_state_bytes(const lpf_ctx* c) {
  if (!c) return LPF_E_ARG;
  size_t n = sizeof(StateHeader);
  for (const auto& s : state_sections(c)) n += s.bytes;
  return (int64_t)n;
}

int lpf_export_state(lpf_ctx* c, void* h_buf, int64_t bytes) {
  if (!c || !h_buf || bytes < lpf_state_bytes(c)) return LPF_E_ARG;
  LPF_CUDA(cudaDeviceSynchronize());
  StateHeader h{};
  memcpy(h.magic, "LPFSTATE", 8);
  h.version = 1; h.params_bytes = (int32_t)sizeof(lpf_params); h.N = c->N; h.total = lpf_state_bytes(c); h.p = c->p;
  char* o = static_cast<char*>(h_buf);
  memcpy(o, &h, sizeof(h)); o += sizeof(h);
  for (const auto& s : state_sections(c)) {
    LPF_CUDA(cudaMemcpy(o, s.d, s.bytes, cudaMemcpyDeviceToHost));
    o += s.bytes;
  }
  return LPF_OK;
}

int lpf_import_state(lpf_ctx* c, const void* h_buf, int64_t bytes) {
  if (!c || !h_buf || bytes < (int64_t)sizeof(StateHeader)) return LPF_E_ARG;
  StateHeader h;
  memcpy(&h, h_buf, sizeof(h));
  if (memcmp(h.magic, "LPFSTATE", 8) != 0 || h.version != 1 || h.params_bytes != (int32_t)sizeof(lpf_params) || h.N != c->N ||
      h.total != lpf_state_bytes(c) || bytes < h.total || memcmp(&h.p, &c->p, sizeof(lpf_params)) != 0)
    return LPF_E_ARG;
  LPF_CUDA(cudaDeviceSynchronize());
  const char* o = static_cast<const char*>(h_buf) + sizeof(h);
  for (const auto& s : state_sections(c)) {
    LPF_CUDA(cudaMemcpy(s.d, o, s.bytes, cudaMemcpyHostToDevice));
    o += s.bytes;
  }
  LPF_CUDA(cudaDeviceSynchronize());
  return LPF_OK;
}

int lpf_destroy(lpf_ctx* c) {
  if (!c) return LPF_E_ARG;
  cudaDeviceSynchronize();
  for (auto& L : c->lanes) free_lane(L);
  void* ptrs[] = {c->W, c->norm_mf, c->norm_bg, c->active, c->forced, c->cpix, c->miss, c->born, c->matched_t,
                  c->slotmap, c->free_list, c->ring, c->meta_t, c->meta_ok, c->counters, c->cube_cache, c->cache_ok,
                  c->cache_t, c->rq_m, c->rq_v, c->rq_state};
  for (void* q : ptrs) if (q) cudaFree(q);
  if (c->ring_ev) cudaEventDestroy(c->ring_ev);
  if (c->chain_st) cudaStreamDestroy(c->chain_st);
  if (c->cap_st) cudaStreamDestroy(c->cap_st);
  if (c->rq_ev) cudaEventDestroy(c->rq_ev);
  lpf_fused_plan_free(c->fused);
  for (cudaEvent_t e : c->prof_pool) cudaEventDestroy(e);
  delete c;
  return LPF_OK;
}

int lpf_cube_qc(lpf_ctx* c, int lane, const float* d_cube, int64_t t, float* d_stats, uint8_t* d_band_ok, void* stream) {
  (void)t;
  TRY(lane_ok(c, lane));
  if (!d_cube || !d_stats || !d_band_ok) return LPF_E_ARG;
  return lpf_launch_qc(c, c->lanes[lane], d_cube, d_stats, d_band_ok, (cudaStream_t)stream);
}

int lpf_detect_sources(lpf_ctx* c, int lane, const float* d_cube, const uint8_t* d_band_ok, lpf_det* d_dets,
                       int32_t* d_ndets, int32_t* d_upos, int16_t* d_uplane, float* d_usnr, int32_t* d_nu, void* stream) {
  TRY(lane_ok(c, lane));
  if (!d_cube || !d_band_ok || !d_dets || !d_ndets || !d_upos || !d_uplane || !d_usnr || !d_nu) return LPF_E_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  LpfLane& L = c->lanes[lane];
  TRY(lpf_launch_detect(c, L, d_cube, d_band_ok, d_dets, d_ndets, false, st));
  return lpf_launch_dedupe(c, L, d_dets, d_ndets, d_upos, d_uplane, d_usnr, d_nu, st);
}

int lpf_associate(lpf_ctx* c, int lane, const int32_t* d_upos, const int32_t* d_nu, const uint8_t* d_band_ok, int64_t t,
                  int32_t* d_cand_idx, int32_t* d_act_slots, int32_t* d_act_pix, int32_t* d_npos, void* stream) {
  TRY(lane_ok(c, lane));
  if (!d_upos || !d_nu || !d_band_ok || !d_cand_idx || !d_act_slots || !d_act_pix || !d_npos || t < 0) return LPF_E_ARG;
  return lpf_launch_associate(c, d_upos, d_nu, d_band_ok, (long long)t, d_cand_idx, d_act_slots, d_act_pix, d_npos,
                              (cudaStream_t)stream);
}

int lpf_add_candidates(lpf_ctx* c, const int32_t* d_pix, int32_t n, int32_t* d_slots_out, void* stream) {
  if (!c || n < 0 || (n > 0 && !d_pix)) return LPF_E_ARG;
  if (n == 0) return LPF_OK;
  if (n > c->p.n_cand_max) return LPF_E_STATE;
  LPF_CUDA(cudaDeviceSynchronize());      // the table is shared with every frame in flight, on every stream
  return lpf_launch_add_candidates(c, d_pix, n, d_slots_out, (cudaStream_t)stream);
}

int lpf_measure_flux(lpf_ctx* c, const float* d_cube, const uint8_t* d_band_ok, const int32_t* d_pos,
                     const int32_t* d_npos, float* d_flux, void* stream) {
  if (!c || !d_cube || !d_band_ok || !d_pos || !d_npos || !d_flux) return LPF_E_ARG;
  return lpf_launch_measure_flux(c, d_cube, d_band_ok, d_pos, d_npos, d_flux, (cudaStream_t)stream);
}

int lpf_append_dynspec(lpf_ctx* c, const int32_t* d_slots, const int32_t* d_n, const float* d_flux,
                       const uint8_t* d_band_ok, int64_t t, void* stream) {
  if (!c || !d_slots || !d_n || !d_flux || !d_band_ok || t < 0) return LPF_E_ARG;
  return lpf_launch_append(c, d_slots, d_n, d_flux, d_band_ok, (long long)t, (cudaStream_t)stream);
}

int lpf_get_dynspec(lpf_ctx* c, int32_t slot, int64_t t_last, float* d_out, void* stream) {
  if (!c || !d_out || slot < 0 || slot >= c->p.n_cand_max) return LPF_E_ARG;
  return lpf_launch_get_dynspec(c, slot, (long long)t_last, d_out, (cudaStream_t)stream);
}

int lpf_export_dynspec(lpf_ctx* c, const int32_t* d_slots, int32_t n, int64_t t_last, const float* d_sigma, float* d_out,
                       void* stream) {
  if (!c || n < 0 || (n > 0 && (!d_slots || !d_out))) return LPF_E_ARG;
  if (n == 0) return LPF_OK;
  return lpf_launch_export_dynspec(c, d_slots, n, (long long)t_last, d_sigma, d_out, (cudaStream_t)stream);
}

int lpf_simulate_pulses(int32_t n, int32_t B, int32_t T, const float* d_nu, float nu0, float dt_s, const float* d_theta,
                        float* d_out, int32_t accumulate, void* stream) {
  if (n < 0 || B < 1 || T < 1 || !(nu0 > 0) || !(dt_s > 0) || (n > 0 && (!d_nu || !d_theta || !d_out))) return LPF_E_ARG;
  if (n == 0) return LPF_OK;
  return lpf_launch_simulate_pulses(n, B, T, d_nu, nu0, dt_s, d_theta, d_out, accumulate, (cudaStream_t)stream);
}

int lpf_process_frame(lpf_ctx* c, int lane, const float* d_cube, int64_t t, void* stream) {
  TRY(lane_ok(c, lane));
  if (!d_cube || t < 0) return LPF_E_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  LpfLane& L = c->lanes[lane];
  // The lane's chain as two CUDA graphs around the association step: one launch instead of nine, one instead of
  // two (a frame then costs the host a third of the time, which is what fills the pipeline after a pause).  For
  // the configuration the graphs were captured for: the fused detection path on an aligned cube, no running
  // per-pixel QC (its state is ordered across lanes by an event), no backward fill (a device-to-device copy of the
  // cube whose source changes per frame), no per-kernel profile.
  const bool graphable = c->fused && (((uintptr_t)d_cube) & 15) == 0 && (c->N & 3) == 0 && !(c->p.zeta_thr > 0) &&
                         c->p.n_back == 0 && !c->prof_on && !L.g_failed;
  if (graphable && !L.gx_a) TRY(build_lane_graphs(c, L, d_cube, (long long)t));
  const bool use_graph = graphable && L.gx_a && L.gx_b;
  if (use_graph) {
    LpfFrameDesc* fd = L.fdesc;
    const float* cube = d_cube;
    long long tt = (long long)t;
    int seq = seq_of(tt);
    void* kargs[4] = {&fd, &cube, &tt, &seq};
    cudaKernelNodeParams kp{};
    kp.func = (void*)k_set_frame; kp.gridDim = dim3(1); kp.blockDim = dim3(1); kp.sharedMemBytes = 0;
    kp.kernelParams = kargs; kp.extra = nullptr;
    LPF_CUDA(cudaGraphExecKernelNodeSetParams(L.gx_a, L.gnode_set, &kp));
    LPF_CUDA(cudaGraphLaunch(L.gx_a, st));
    c->launches += L.g_nodes_a;
  } else {
    TRY(lpf_launch_qc_sum(c, L, d_cube, L.stats, L.band_ok, L.ndets, st));      // S1-S3
    if (c->p.n_back > 0) TRY(lpf_launch_cache_store(c, d_cube, L.band_ok, (long long)t, st));   // O11: the frame joins the cache
    TRY(lpf_launch_detect(c, L, d_cube, L.band_ok, L.dets, L.ndets, true, st));
    TRY(lpf_launch_dedupe(c, L, L.dets, L.ndets, L.upos, L.uplane, L.usnr, L.nu, st));
  }
  // The candidate table and the rings are shared by all lanes.  The association steps of all frames run, in frame
  // order, on ONE stream of the context (highest priority: a single block per frame that the next frame waits for
  // must not queue behind the other lanes' grids); the lane's stream hands over after its duplicate filter and
  // takes over again for the flux measurement.  The ring steps are ordered across lanes by an event (a slot born
  // at t is blanked by the append of frame t, which must not follow the append of frame t + 1); they do not hold
  // up the association of frame t + 1.
  LPF_CUDA(cudaEventRecord(L.ev_pre, st));
  LPF_CUDA(cudaStreamWaitEvent(c->chain_st, L.ev_pre, 0));
  TRY(lpf_launch_associate(c, L.upos, L.nu, L.band_ok, (long long)t, L.cand_idx, L.act_slots, L.act_pix, L.npos, c->chain_st));
  LPF_CUDA(cudaEventRecord(L.ev_post, c->chain_st));
  LPF_CUDA(cudaStreamWaitEvent(st, L.ev_post, 0));
  if (c->ring_valid) LPF_CUDA(cudaStreamWaitEvent(st, c->ring_ev, 0));
  if (use_graph) {
    LPF_CUDA(cudaGraphLaunch(L.gx_b, st));
    c->launches += L.g_nodes_b;
  } else {
    TRY(lpf_launch_measure_flux(c, d_cube, L.band_ok, L.act_pix, L.npos, L.flux, st));
    TRY(lpf_launch_append(c, L.act_slots, L.npos, L.flux, L.band_ok, (long long)t, st));
    if (c->p.n_back > 0) TRY(lpf_launch_backfill(c, L.act_slots, L.act_pix, L.npos, d_cube, L.band_ok, (long long)t, st));   // O11
  }
  LPF_CUDA(cudaEventRecord(c->ring_ev, st));
  c->ring_valid = true;
  return LPF_OK;
}

int lpf_get_frame_view(lpf_ctx* c, int lane, lpf_frame_view* v) {
  TRY(lane_ok(c, lane));
  if (!v) return LPF_E_ARG;
  const LpfLane& L = c->lanes[lane];
  v->d_stats = L.stats; v->d_band_ok = L.band_ok; v->d_dets = L.dets; v->d_ndets = L.ndets;
  v->d_upos = L.upos; v->d_uplane = L.uplane; v->d_usnr = L.usnr; v->d_nu = L.nu; v->d_cand_idx = L.cand_idx;
  v->d_act_slots = L.act_slots; v->d_act_pix = L.act_pix; v->d_npos = L.npos; v->d_flux = L.flux;
  v->d_zeta_cnt = L.zeta_cnt;
  return LPF_OK;
}

int lpf_process_frame_host_begin(lpf_ctx* c, int lane, const float* h_cube, int64_t t, lpf_host_result* res, void* stream) {
  TRY(lane_ok(c, lane));
  if (!h_cube || !res) return LPF_E_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  LpfLane& L = c->lanes[lane];
  const lpf_params& p = c->p;
  const size_t cube_bytes = (size_t)p.B * c->N * sizeof(float);
  if (!L.cube) TRY(dalloc(&L.cube, (size_t)p.B * c->N));
  LPF_CUDA(cudaMemcpyAsync(L.cube, h_cube, cube_bytes, cudaMemcpyHostToDevice, st));
  TRY(lpf_process_frame(c, lane, L.cube, t, st));
  LPF_CUDA(cudaMemcpyAsync(&L.h_counts[0], L.nu, 4, cudaMemcpyDeviceToHost, st));
  LPF_CUDA(cudaMemcpyAsync(&L.h_counts[1], L.npos, 4, cudaMemcpyDeviceToHost, st));
  LPF_CUDA(cudaMemcpyAsync(&L.h_counts[2], L.ndets, 4, cudaMemcpyDeviceToHost, st));
  if (res->h_stats) LPF_CUDA(cudaMemcpyAsync(res->h_stats, L.stats, (size_t)p.B * LPF_STATS_PER_BAND * 4, cudaMemcpyDeviceToHost, st));
  if (res->h_band_ok) LPF_CUDA(cudaMemcpyAsync(res->h_band_ok, L.band_ok, (size_t)p.B + 1, cudaMemcpyDeviceToHost, st));
  return LPF_OK;
}

int lpf_process_frame_host_end(lpf_ctx* c, int lane, lpf_host_result* res, void* stream) {
  TRY(lane_ok(c, lane));
  if (!res) return LPF_E_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  LpfLane& L = c->lanes[lane];
  const lpf_params& p = c->p;
  LPF_CUDA(cudaStreamSynchronize(st));
  res->nu = L.h_counts[0]; res->npos = L.h_counts[1]; res->ndets = L.h_counts[2];
  const int cap_u = res->cap_u > 0 ? res->cap_u : 0, cap_pos = res->cap_pos > 0 ? res->cap_pos : 0;
  const size_t nu = (size_t)(res->nu < cap_u ? res->nu : cap_u);
  const size_t np = (size_t)(res->npos < cap_pos ? res->npos : cap_pos);
  const bool truncated = res->ndets > p.max_det || res->nu > cap_u || res->npos > cap_pos;
  if (nu) {
    if (res->h_upos) LPF_CUDA(cudaMemcpyAsync(res->h_upos, L.upos, nu * 4, cudaMemcpyDeviceToHost, st));
    if (res->h_uplane) LPF_CUDA(cudaMemcpyAsync(res->h_uplane, L.uplane, nu * 2, cudaMemcpyDeviceToHost, st));
    if (res->h_usnr) LPF_CUDA(cudaMemcpyAsync(res->h_usnr, L.usnr, nu * 4, cudaMemcpyDeviceToHost, st));
    if (res->h_cand_idx) LPF_CUDA(cudaMemcpyAsync(res->h_cand_idx, L.cand_idx, nu * 4, cudaMemcpyDeviceToHost, st));
  }
  if (np) {
    if (res->h_act_slots) LPF_CUDA(cudaMemcpyAsync(res->h_act_slots, L.act_slots, np * 4, cudaMemcpyDeviceToHost, st));
    if (res->h_flux) LPF_CUDA(cudaMemcpyAsync(res->h_flux, L.flux, np * p.B * 4, cudaMemcpyDeviceToHost, st));
  }
  LPF_CUDA(cudaStreamSynchronize(st));
  return truncated ? LPF_W_CAPACITY : LPF_OK;
}

int lpf_process_frame_host(lpf_ctx* c, int lane, const float* h_cube, int64_t t, lpf_host_result* res, void* stream) {
  TRY(lpf_process_frame_host_begin(c, lane, h_cube, t, res, stream));
  return lpf_process_frame_host_end(c, lane, res, stream);
}

int lpf_get_counters(lpf_ctx* c, int64_t* h_out) {
  if (!c || !h_out) return LPF_E_ARG;
  int32_t h[4];
  LPF_CUDA(cudaDeviceSynchronize());
  LPF_CUDA(cudaMemcpy(h, c->counters, sizeof(h), cudaMemcpyDeviceToHost));
  h_out[0] = h[0]; h_out[1] = h[1]; h_out[2] = c->launches; h_out[3] = h[2];
  return (h[0] > 0 || h[1] > 0) ? LPF_W_CAPACITY : LPF_OK;
}

static const char* const kKernelNames[KID_COUNT] = {
    "qc_pass1", "qc_pass2", "qc_running", "sum_plane", "conv_mf", "conv_c", "conv_s", "conv_den", "threshold_peaks",
    "fused_detect", "dedupe_scatter", "dedupe_select", "dedupe_sort", "assoc_match", "assoc_update", "measure_flux",
    "append_dynspec", "backfill", "misc", "peaks", "qc_verdict", "qc_clip_finish"};

int lpf_profile_begin(lpf_ctx* c) {
  if (!c) return LPF_E_ARG;
  LPF_CUDA(cudaDeviceSynchronize());
  c->prof_recs.clear();
  c->prof_pool_used = 0;
  c->prof_on = true;
  return LPF_OK;
}

int lpf_profile_end(lpf_ctx* c, int32_t* h_count, float* h_ms, int32_t n) {
  if (!c || !h_count || !h_ms || n < KID_COUNT) return LPF_E_ARG;
  c->prof_on = false;
  LPF_CUDA(cudaDeviceSynchronize());
  for (int i = 0; i < n; ++i) { h_count[i] = 0; h_ms[i] = 0.f; }
  for (const auto& r : c->prof_recs) {
    float ms = 0.f;
    LPF_CUDA(cudaEventElapsedTime(&ms, r.e0, r.e1));
    h_count[r.kid] += 1; h_ms[r.kid] += ms;
  }
  c->prof_recs.clear();
  c->prof_pool_used = 0;
  return LPF_OK;
}

int lpf_profile_timeline(lpf_ctx* c, int32_t* h_kid, float* h_t0_ms, float* h_t1_ms, int32_t n_max) {
  if (!c || !h_kid || !h_t0_ms || !h_t1_ms || n_max < 0) return LPF_E_ARG;
  c->prof_on = false;
  LPF_CUDA(cudaDeviceSynchronize());
  int n = 0;
  for (const auto& r : c->prof_recs) {
    if (n >= n_max) break;
    float a = 0.f, b = 0.f;
    LPF_CUDA(cudaEventElapsedTime(&a, c->prof_recs.front().e0, r.e0));
    LPF_CUDA(cudaEventElapsedTime(&b, c->prof_recs.front().e0, r.e1));
    h_kid[n] = r.kid; h_t0_ms[n] = a; h_t1_ms[n] = b; ++n;
  }
  c->prof_recs.clear();
  c->prof_pool_used = 0;
  return n;
}

int lpf_get_plan(lpf_ctx* c, int64_t* h_out) {
  if (!c || !h_out) return LPF_E_ARG;
  int cw = 0, th = 0, ni = 0; long long sm = 0;
  h_out[0] = lpf_fused_plan_info(c->fused, &cw, &th, &ni, &sm);
  h_out[1] = cw; h_out[2] = th; h_out[3] = ni; h_out[4] = sm; h_out[5] = c->n_planes; h_out[6] = c->n_sm; h_out[7] = c->qc_nblk;
  return LPF_OK;
}

int lpf_profile_kernel_count(void) { return KID_COUNT; }
const char* lpf_profile_kernel_name(int kid) { return (kid >= 0 && kid < KID_COUNT) ? kKernelNames[kid] : ""; }

int lpf_memcpy_d2h(void* h_dst, const void* d_src, int64_t bytes) {
  if (bytes < 0 || (bytes > 0 && (!h_dst || !d_src))) return LPF_E_ARG;
  if (bytes == 0) return LPF_OK;
  LPF_CUDA(cudaMemcpy(h_dst, d_src, (size_t)bytes, cudaMemcpyDeviceToHost));
  return LPF_OK;
}

const char* lpf_strerror(int code) {
  switch (code) {
    case LPF_OK: return "ok";
    case LPF_E_ARG: return "bad argument or unsupported parameter";
    case LPF_E_CUDA: return "CUDA runtime error";
    case LPF_E_STATE: return "bad state (call order, capacity)";
    case LPF_E_NOMEM: return "out of device memory";
    case LPF_E_TOO_LARGE: return "the problem exceeds a fixed maximum of this entry point";
    case LPF_W_CAPACITY: return "warning: a list was truncated (capacity); the dropped entries are counted";
    default: return "unknown";
  }
}

const char* lpf_last_cuda_error(void) { return g_lpf_cuda_err; }

int lpf_version(void) { return 100; }

}  // extern "C"
