// Internal declarations of the LPF CUDA library (sm_100a).  Not part of the C-ABI.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <vector>

#include "../../include/lpf.h"

#define LPF_NTAPS (2 * LPF_MAX_RADIUS + 1)

struct LpfTaps {
  int R;
  float g[LPF_NTAPS];
};

// What changes from one frame to the next on a lane.  With the lane's frame chain captured in CUDA graphs the kernels
// read it from device memory (written by the first node of the graph, the one node whose parameters are updated per
// launch); launched directly they get the same values in their arguments (fd = null).
struct LpfFrameDesc { const float* cube; long long t; int32_t seq; int32_t pad; };

// Scratch and owned outputs of one frame in flight.
struct LpfLane {
  double* qc_part1 = nullptr;  // [B][nblk][3]  n, sum(x-p), sum(x-p)^2
  double* qc_part2 = nullptr;  // [blocks of pass 2][B][3]  clipped
  float* qc_band_clip = nullptr;   // [B][2] centre, half width of the clip round
  int32_t* qc_counter = nullptr;   // [2] last-block counters of the two passes
  double* qc_mom = nullptr;        // [B][3] finished sums of the streaming QC
  float* sum_plane = nullptr;  // [N]
  int32_t* dirty = nullptr;    // [1] == dirty_seq: the cube of the current frame needs masking (detect_general.cu k_sum_plane)
  int32_t dirty_seq = 0;
  int32_t* dirty_b = nullptr;  // [B] == dirty_seq: that band is not an exact zero at some invalid pixel (streaming QC)
  float* F = nullptr;          // [(B+1)][N] matched-filtered planes (general path)
  float* C = nullptr;          // [(B+1)][N]
  float* S = nullptr;          // [(B+1)][N]
  uint8_t* Y = nullptr;        // [(B+1)][N] iteration of first detection (n_iter > 1 only)
  float* normp = nullptr;      // [(B+1)][N] per-plane normaliser for iterations > 1
  unsigned long long* M = nullptr;  // [N] dedupe key map, all zero between frames
  int32_t* tmp_pos = nullptr;
  int16_t* tmp_plane = nullptr;
  float* tmp_snr = nullptr;
  int32_t* tmp_n = nullptr;
  // lane-owned results of lpf_process_frame
  float* stats = nullptr;
  uint8_t* band_ok = nullptr;
  lpf_det* dets = nullptr;
  int32_t* ndets = nullptr;
  int32_t* upos = nullptr;
  int16_t* uplane = nullptr;
  float* usnr = nullptr;
  int32_t* nu = nullptr;
  int32_t* cand_idx = nullptr;
  int32_t* act_slots = nullptr;
  int32_t* act_pix = nullptr;
  int32_t* npos = nullptr;
  float* flux = nullptr;
  float* cube = nullptr;       // device cube for the *_host entry (lazy)
  int32_t* zeta_cnt = nullptr; // [B] eq. A.2 counts of the lane's frame
  void* hits = nullptr;        // fused path: the hit list of the frame, [segments][seg_cap] entries (detect_fused.cu)
  int32_t* hit_cnt = nullptr;  // [segments]
  float* big_thr = nullptr;    // [B + 1] 'far above the noise' level of every plane (64 x rms)
  int32_t* h_counts = nullptr; // pinned [4]
  cudaEvent_t ev_pre = nullptr, ev_post = nullptr;   // hand-over to / from the context's association stream
  // the lane's frame chain as two CUDA graphs (before / after the association step), built on first use
  LpfFrameDesc* fdesc = nullptr;       // device
  cudaGraph_t g_a = nullptr;
  cudaGraphExec_t gx_a = nullptr, gx_b = nullptr;
  cudaGraphNode_t gnode_set = nullptr; // the k_set_frame node of gx_a
  int g_nodes_a = 0, g_nodes_b = 0;
  bool g_failed = false;               // capture was refused once: the lane launches its kernels directly
};

struct LpfFusedPlan;  // detect_fused.cu

struct lpf_ctx {
  LpfFusedPlan* fused = nullptr;  // non-null: the fused fast path serves lpf_detect_sources
  lpf_params p;
  int64_t N;        // Dy*Dx
  int n_planes;     // B + detect_sum_plane
  int qc_nblk;
  int first_valid;  // first valid pixel (pivot of the statistics)
  int n_sm;
  LpfTaps g_mf, g_bg;
  uint8_t* W = nullptr;      // [N] valid mask (always materialised)
  float* norm_mf = nullptr;  // [N] W / (g_mf (*) W)
  float* norm_bg = nullptr;  // [N] W / (g_bg (*) W)
  // candidate table
  uint8_t* active = nullptr;
  uint8_t* forced = nullptr;
  int32_t* cpix = nullptr;
  int32_t* miss = nullptr;
  long long* born = nullptr;
  long long* matched_t = nullptr;
  int32_t* slotmap = nullptr;  // [N] lowest active slot at that pixel, -1 none
  int32_t* free_list = nullptr;
  float* ring = nullptr;       // [n_cand_max][T_ring][B]
  long long* meta_t = nullptr; // [T_ring]
  unsigned long long* meta_ok = nullptr;
  int32_t* counters = nullptr; // [0] dropped records, [1] dropped detections, [2] active candidates
  // running per-pixel QC (O12, eq. A.2): two copies of the mean / variance images (the update of a frame is written
  // to the other copy and adopted per band only if the band is accepted), update counts, scratch
  float* rq_m = nullptr;            // [2][B][N]
  float* rq_v = nullptr;            // [2][B][N]
  int32_t* rq_state = nullptr;      // [B] current copy, [B] updates so far, [B] counts of the frame in progress, [B] consecutive discards, [1] block counter
  cudaEvent_t rq_ev = nullptr;      // orders the frames' updates across lanes
  bool rq_valid = false;
  // backward fill (O11): the last n_back cubes, their verdicts and time steps
  float* cube_cache = nullptr;      // [n_back + n_lanes][B][N]
  uint8_t* cache_ok = nullptr;      // [n_back + n_lanes][B + 1]
  long long* cache_t = nullptr;     // [n_back + n_lanes], -1 = empty
  cudaStream_t cap_st = nullptr;    // stream the lanes' graphs are captured on
  const LpfFrameDesc* cap_fd = nullptr;   // non-null while a capture is in progress: the launchers point the kernels at it
  cudaStream_t chain_st = nullptr;  // the association steps of all frames, in frame order (highest priority)
  cudaEvent_t ring_ev = nullptr;    // after the ring steps (append, backward fill) of the latest frame
  bool ring_valid = false;
  int64_t launches = 0;
  std::vector<LpfLane> lanes;
  // per-kernel profile
  bool prof_on = false;
  struct ProfRec { int kid; cudaEvent_t e0, e1; };
  std::vector<ProfRec> prof_recs;
  std::vector<cudaEvent_t> prof_pool;
  size_t prof_pool_used = 0;
};

extern thread_local char g_lpf_cuda_err[256];
int lpf_cuda_fail(cudaError_t e, const char* what);

#define LPF_CUDA(call)                                        \
  do {                                                        \
    cudaError_t e__ = (call);                                 \
    if (e__ != cudaSuccess) return lpf_cuda_fail(e__, #call); \
  } while (0)

// Kernel ids for the optional per-kernel CUDA-event profile (lpf_profile_begin / lpf_profile_end).
enum LpfKernelId {
  KID_QC_PASS1 = 0, KID_QC_PASS2, KID_QC_VERDICT /* = the running per-pixel test, eq. A.2 */, KID_SUM_PLANE, KID_CONV_MF, KID_CONV_C, KID_CONV_S,
  KID_CONV_DEN, KID_THRESHOLD, KID_FUSED_DETECT, KID_DEDUPE_SCATTER, KID_DEDUPE_SELECT, KID_DEDUPE_SORT,
  KID_ASSOC_MATCH, KID_ASSOC_UPDATE, KID_MEASURE_FLUX, KID_APPEND, KID_BACKFILL, KID_MISC, KID_PEAKS, KID_QC_VERDICT1, KID_QC_CLIPFIN, KID_COUNT
};
void lpf_prof_pre(lpf_ctx* c, int kid, cudaStream_t st);
void lpf_prof_post(lpf_ctx* c, cudaStream_t st);

// Launch `...` (a kernel<<<>>>() expression) on stream st, count it, bracket it with events when profiling.
#define LPF_KLAUNCH(ctx, kid, st, ...)                             \
  do {                                                            \
    if ((ctx)->prof_on) lpf_prof_pre((ctx), (kid), (st));         \
    __VA_ARGS__;                                                  \
    if ((ctx)->prof_on) lpf_prof_post((ctx), (st));               \
    (ctx)->launches++;                                            \
    cudaError_t e__ = cudaPeekAtLastError();                      \
    if (e__ != cudaSuccess) return lpf_cuda_fail(e__, #kid);      \
  } while (0)

// ---- launchers implemented in the kernel translation units ---------------------------------
int lpf_launch_qc(lpf_ctx* c, LpfLane& L, const float* d_cube, float* d_stats, uint8_t* d_band_ok, cudaStream_t st);
int lpf_launch_qc_sum(lpf_ctx* c, LpfLane& L, const float* d_cube, float* d_stats, uint8_t* d_band_ok, int32_t* zero_me,
                      cudaStream_t st);
int lpf_qc2_blocks(const lpf_ctx* c);
int lpf_qs_blocks(const lpf_ctx* c);
int lpf_qc_prepare(void);
int lpf_general_prepare(void);
int lpf_launch_qc_running(lpf_ctx* c, LpfLane& L, const float* d_cube, uint8_t* d_band_ok, cudaStream_t st);

int lpf_launch_sum_plane(lpf_ctx* c, LpfLane& L, const float* d_cube, const uint8_t* d_band_ok, bool want_sum, cudaStream_t st);
int lpf_launch_detect_general(lpf_ctx* c, LpfLane& L, const float* d_cube, const uint8_t* d_band_ok,
                              lpf_det* d_dets, int32_t* d_ndets, bool sum_done, cudaStream_t st);
int lpf_fused_plan(lpf_ctx* c, const uint8_t* hW, LpfFusedPlan** out);
void lpf_fused_plan_free(LpfFusedPlan* pl);
int lpf_fused_plan_info(const LpfFusedPlan* pl, int* cw, int* threads, int* n_items, long long* smem);
void lpf_fused_hit_sizes(const LpfFusedPlan* pl, int n_planes, long long* hit_bytes, long long* n_seg);
float lpf_fused_big_sigma(void);
int lpf_launch_detect_fused(lpf_ctx* c, LpfFusedPlan* pl, LpfLane& L, const float* d_cube, const uint8_t* d_band_ok,
                            lpf_det* d_dets, int32_t* d_ndets, bool sum_done, cudaStream_t st);
int lpf_launch_detect(lpf_ctx* c, LpfLane& L, const float* d_cube, const uint8_t* d_band_ok, lpf_det* d_dets,
                      int32_t* d_ndets, bool sum_done, cudaStream_t st);
int lpf_ensure_general_scratch(lpf_ctx* c, LpfLane& L);
int lpf_launch_static_norm(lpf_ctx* c, const LpfTaps& g, float* d_norm, float* d_tmp, cudaStream_t st);

int lpf_launch_dedupe(lpf_ctx* c, LpfLane& L, const lpf_det* d_dets, const int32_t* d_ndets, int32_t* d_upos,
                      int16_t* d_uplane, float* d_usnr, int32_t* d_nu, cudaStream_t st);
int lpf_launch_associate(lpf_ctx* c, const int32_t* d_upos, const int32_t* d_nu, const uint8_t* d_band_ok,
                         long long t, int32_t* d_cand_idx, int32_t* d_act_slots, int32_t* d_act_pix,
                         int32_t* d_npos, cudaStream_t st);
int lpf_launch_add_candidates(lpf_ctx* c, const int32_t* d_pix, int n, int32_t* d_slots_out, cudaStream_t st);
int lpf_launch_measure_flux(lpf_ctx* c, const float* d_cube, const uint8_t* d_band_ok, const int32_t* d_pos,
                            const int32_t* d_npos, float* d_flux, cudaStream_t st);
int lpf_launch_append(lpf_ctx* c, const int32_t* d_slots, const int32_t* d_n, const float* d_flux,
                      const uint8_t* d_band_ok, long long t, cudaStream_t st);
int lpf_launch_backfill(lpf_ctx* c, const int32_t* d_slots, const int32_t* d_pix, const int32_t* d_n, const float* d_cube,
                        const uint8_t* d_band_ok, long long t, cudaStream_t st);
int lpf_launch_export_dynspec(lpf_ctx* c, const int32_t* d_slots, int n, long long t_last, const float* d_sigma, float* d_out,
                              cudaStream_t st);
int lpf_launch_simulate_pulses(int n, int B, int T, const float* d_nu, float nu0, float dt_s, const float* d_theta, float* d_out,
                               int accumulate, cudaStream_t st);
int lpf_launch_cache_store(lpf_ctx* c, const float* d_cube, const uint8_t* d_band_ok, long long t, cudaStream_t st);
int lpf_launch_get_dynspec(lpf_ctx* c, int slot, long long t_last, float* d_out, cudaStream_t st);
int lpf_launch_fill_nan(lpf_ctx* c, float* d, int64_t n, cudaStream_t st);
int lpf_launch_fill_i32(lpf_ctx* c, int32_t* d, int64_t n, int32_t v, cudaStream_t st);

// ---- small device helpers --------------------------------------------------------------------
__device__ __forceinline__ float lpf_warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ double lpf_warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ int lpf_warp_sum(int v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
