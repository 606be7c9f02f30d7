/* lpf.h -- C-ABI of the B200-native LPF hot path ("Live Pulse Finder").
 *
 * The per-time-step source-detection and flux-measurement stage of Ruhe et al.,
 * arXiv 2103.15418, over a streaming image cube X_t in R^{B x D x D}:
 *
 *   lpf_cube_qc        quality control            App. A, eq. A.1
 *   lpf_detect_sources peak detection/localisation  eqs. 2-7
 *                      + cross-frequency duplicate filter
 *   lpf_associate      match to the t-1 catalogue, monitoring
 *   lpf_measure_flux   max pixel in a box, all frequencies
 *   lpf_append_dynspec dynamic spectra (frequency x time)           (Fig. 1 :23)
 *
 * Conventions
 *   - Every pointer named d_* is DEVICE memory (sm_100a, one GPU); h_* is HOST
 *     memory.  The caller owns the cube and every output buffer; the context owns
 *     its scratch (one set per lane), the candidate table, the slot map and the
 *     rings.  The cube is never written (a rejected band is expressed by band_ok).
 *   - `stream` is a cudaStream_t passed as void*.  Every call only enqueues work
 *     on it; counts live in device memory; nothing on the hot path synchronises
 *     with the host (lpf_create, lpf_destroy, lpf_get_counters and the *_host
 *     entry point do).
 *   - Layout: cube [B][Dy][Dx] float32, x fastest; pix = y*Dx + x; plane p < B is
 *     band p, plane B is the sum over accepted bands.
 *   - lpf_associate / lpf_append_dynspec must be issued in increasing t.  A lane
 *     (0 <= lane < n_lanes) is a set of scratch buffers; two frames in flight at
 *     the same time must use different lanes (BASELINE.json config 4: 4 lanes).
 *   - Return value: 0 = LPF_OK; negative = error (nothing was enqueued); positive = warning (LPF_W_CAPACITY,
 *     reported at the sync points lpf_get_counters and lpf_process_frame_host / _host_end).
 *     Capacity overflow (max_det, n_cand_max) is not undefined behaviour: the list
 *     is truncated and a device counter is incremented (lpf_get_counters).
 *   - There is no CPU fallback: without a CUDA device lpf_create returns
 *     LPF_E_CUDA.
 *
 * Definitions O1..O10 and readings R1..R24 referenced below are in DESIGN.md.
 */
#ifndef LPF_H_
#define LPF_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LPF_OK 0
#define LPF_E_ARG (-1)   /* bad argument / unsupported parameter value */
#define LPF_E_CUDA (-2)  /* a CUDA runtime call failed (see lpf_last_cuda_error) */
#define LPF_E_STATE (-3) /* call order / lane misuse */
#define LPF_E_NOMEM (-4)
#define LPF_E_TOO_LARGE (-5) /* the problem exceeds a fixed maximum of the entry point (lpf_last_cuda_error says which) */
#define LPF_W_CAPACITY 1  /* positive = warning, the call did its work: a list was truncated (max_det, n_cand_max, the
                           * hit list of the fused path, or a caller buffer); the dropped entries are counted */

#define LPF_MAX_BANDS 64  /* band_ok bits are kept in one 64-bit word per time step */
#define LPF_MAX_RADIUS 16 /* k_mf, k_bg <= 16 ; k_max, r_flux, r_dedupe, r_assoc <= 8 */
#define LPF_STATS_PER_BAND 8

typedef struct lpf_ctx lpf_ctx; /* opaque */

/* Plain-old-data parameter block, copied at lpf_create. */
typedef struct {
  int32_t B, Dy, Dx;        /* cube shape; 1 <= B <= 64 */
  float kappa;              /* eq. 5 threshold */
  int32_t k_max;            /* eq. 6 max-filter half width (window 2k+1) */
  float eps_rel;            /* rounding guard S_eff = max(S, (eps_rel |C|)^2) (R8); 1e-5 */
  float sigma_mf;           /* matched-filter Gaussian sigma [px]; <= 0: F = X (paper-literal) */
  int32_t k_mf;             /* matched-filter half width */
  int32_t bg_kernel;        /* background kernel G of eqs. 3-4: 0 = Gaussian (eq. 2), 1 = uniform box */
  float s_bg;               /* Gaussian s of eq. 2 (ignored for the box) */
  int32_t k_bg;             /* half width of G */
  int32_t n_iter;           /* sigma-clip iterations, >= 1 */
  int32_t detect_sum_plane; /* also run eqs. 2-7 on the channel-summed plane (north_star; R5) */
  float qc_tau;             /* eq. A.1 threshold, "e.g. 5" */
  float qc_clip;            /* sigma of the one clip round behind the clipped mean/rms (R13) */
  int32_t r_flux;           /* flux box half width (R15) */
  int32_t r_dedupe;         /* duplicate-filter radius [px] (R17) */
  int32_t r_assoc;          /* association radius [px] (R16) */
  int32_t n_forget;         /* retire after this many accepted frames without a detection */
  int32_t T_ring;           /* dynamic-spectrum ring length [time steps] */
  int32_t n_cand_max;       /* candidate-table capacity */
  int32_t max_det;          /* capacity of the per-plane record list, per frame */
  int32_t n_lanes;          /* frames in flight */
  int32_t n_back;           /* backward fill: a slot created at t also gets the fluxes of the last n_back
                             * cubes, which lpf_process_frame then keeps in a device cache; 0 = off, <= 64 */
  float zeta_thr;           /* eq. A.2: per-pixel running mean / variance of every band; a band with more
                             * than zeta_nmax valid pixels (with var > 0) at |x - mean| > zeta_thr * sqrt(var) is discarded; 0 = off */
  int32_t zeta_nmax;        /* 0 = the paper's "if zeta exceeds a threshold" */
  int32_t zeta_window;      /* Welford up to this many updates, exponentially weighted (alpha = 1/window) after */
  int32_t zeta_warm;        /* no test before a band has had this many updates; >= 2 (after one update every variance is 0) */
  int32_t zeta_reset;       /* a band discarded by eq. A.2 in this many consecutive frames starts over (its running state is
                             * forgotten: Welford from scratch, untested during the warm-up) -- the way out of a lasting level
                             * change; 0 = never (a discarded band keeps its state, R22) */
  int32_t force_general;    /* 1: lpf_detect_sources takes the general multi-kernel path even when the parameter set allows the
                             * fused single-pass kernel (used by the parity tests to reach both); 0: automatic */
} lpf_params;

/* One peak (eq. 7: p = q and y) of one plane.  24 bytes. */
typedef struct {
  int32_t pix;   /* y*Dx + x */
  int16_t plane; /* 0..B-1 band, B = sum plane */
  int16_t iter;  /* sigma-clip iteration of first detection, 1-based */
  float f;       /* matched-filtered value F at the peak */
  float c;       /* local centre C (eq. 3) at first detection */
  float s;       /* local spread S_eff (eq. 4 + guard R8) at first detection */
  float snr;     /* (F - C) / sqrt(S_eff) */
} lpf_det;

/* Device-side views of what lpf_process_frame left in a lane (valid until the lane is reused). */
typedef struct {
  const float* d_stats;      /* [B][8] n, mean, rms, n_clip, clipped mean, clipped rms, z_mean, z_rms */
  const uint8_t* d_band_ok;  /* [B+1], last = frame_ok */
  const lpf_det* d_dets;     /* [<= max_det] unordered */
  const int32_t* d_ndets;    /* [1] number of records found (may exceed max_det: truncated) */
  const int32_t* d_upos;     /* unique detections, ascending pix */
  const int16_t* d_uplane;   /* plane of the largest snr at that pixel */
  const float* d_usnr;       /* that snr */
  const int32_t* d_nu;       /* [1] */
  const int32_t* d_cand_idx; /* [nu] candidate slot of each unique detection (-1: dropped / rejected frame) */
  const int32_t* d_act_slots;/* [npos] active slots after this frame, ascending */
  const int32_t* d_act_pix;  /* [npos] their pixels */
  const int32_t* d_npos;     /* [1] */
  const float* d_flux;       /* [npos][B] */
  const int32_t* d_zeta_cnt; /* [B] pixels over the eq. A.2 threshold in this frame (zeros when the test is off) */
} lpf_frame_view;

/* Host-side result sizes / pointers for lpf_process_frame_host (all HOST memory, caller-owned). */
typedef struct {
  float* h_stats;        /* [B][8] */
  uint8_t* h_band_ok;    /* [B+1] */
  int32_t* h_upos;       /* [cap_u] */
  int16_t* h_uplane;     /* [cap_u] */
  float* h_usnr;         /* [cap_u] */
  int32_t* h_cand_idx;   /* [cap_u] */
  int32_t cap_u;         /* capacity of the four arrays above */
  int32_t* h_act_slots;  /* [cap_pos] */
  float* h_flux;         /* [cap_pos][B] */
  int32_t cap_pos;
  int32_t nu, npos, ndets; /* written by the call */
} lpf_host_result;

/* -- life cycle ------------------------------------------------------------ */
/* d_valid_mask: device uint8 [Dy][Dx] (1 = valid pixel W, R7/R14) or NULL (all valid); copied.
 * Synchronises.  Precomputes the static normalised-convolution denominators (R7). */
int lpf_create(lpf_ctx** out, const lpf_params* p, const uint8_t* d_valid_mask);
int lpf_destroy(lpf_ctx* ctx);

/* -- S1+S2: quality control (App. A; O1, O2) --------------------------------
 * d_stats [B][8] float32, d_band_ok [B+1] uint8 (band_ok[B] = frame_ok).
 * Per band over valid pixels: n, mean b (the paper's b), rms, and after one
 * qc_clip-sigma clip round n_clip, clipped mean, clipped rms; then eq. A.1 z-scores of the mean
 * and of the rms across bands (median / median-absolute-deviation, SE floor; R10-R13);
 * band_ok = |z_mean| <= tau and |z_rms| <= tau; frame_ok = #ok >= ceil(B/2).
 * With zeta_thr > 0 the per-pixel running test of eq. A.2 (O12) follows: it can discard further bands (frame_ok is
 * re-evaluated) and advances the running mean / variance images of the bands it accepts, so call it once per cube,
 * in increasing t (the calls of different lanes are ordered by an event). */
int lpf_cube_qc(lpf_ctx* ctx, int lane, const float* d_cube, int64_t t, float* d_stats,
                uint8_t* d_band_ok, void* stream);

/* The same statistics and eq. A.1 verdict (d_stats, d_band_ok as above; no eq. A.2 step, no lane) for callers that
 * cannot reach cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it): the call
 * and everything behind it allocate nothing.  Its scratch (per-block partial sums, clip parameters, two block
 * counters) is a static device array of LPF_QC_STATIC_BYTES that every GPU which loads the library holds until the
 * process exits.  Limit: B x (blocks of the two passes) x 24 bytes + 2 KB must fit (every BASELINE.json
 * configuration does: 1024 x 1024 x 64 needs 0.87 MB); beyond it the call returns LPF_E_TOO_LARGE, launches nothing,
 * and lpf_last_cuda_error names the sizes.  All calls on a device share the array: calls that overlap on the GPU
 * (two streams) race; calls on one stream, or ordered by events, do not.  The first call on a device asks the
 * runtime for the array's device address (cudaGetSymbolAddress): make that call outside a stream capture.
 * Kernels: the generic k_qc_pass1 / k_qc_pass2 (any alignment of d_cube). */
#define LPF_QC_STATIC_BYTES (1 << 20)
int lpf_cube_qc_static(lpf_ctx* ctx, const float* d_cube, float* d_stats, uint8_t* d_band_ok, void* stream);

/* -- S3-S9: detection (eqs. 2-7; O3-O7) -------------------------------------
 * For every accepted plane: F = g_mf (*)_W X; n_iter rounds of C = G (*)_W' F,
 * S = G (*)_W' (F-C)^2, y = [F-C > 0 and (F-C)^2 > kappa^2 S_eff]; q = local max of F over the
 * (2 k_max+1)^2 window; p = q and y.  Records (unordered) go to d_dets / d_ndets; then the
 * cross-plane duplicate filter writes the unique positions sorted by pix.
 * Capacities: d_dets [max_det]; d_upos/d_uplane/d_usnr [max_det].
 * A rejected frame (band_ok[B] = 0) yields ndets = nu = 0. */
int lpf_detect_sources(lpf_ctx* ctx, int lane, const float* d_cube, const uint8_t* d_band_ok,
                       lpf_det* d_dets, int32_t* d_ndets, int32_t* d_upos, int16_t* d_uplane,
                       float* d_usnr, int32_t* d_nu, void* stream);

/* -- S10: association + monitoring (O8) -----------------------
 * d_cand_idx [nu]; d_act_slots / d_act_pix [n_cand_max]; d_npos [1]. */
int lpf_associate(lpf_ctx* ctx, int lane, const int32_t* d_upos, const int32_t* d_nu,
                  const uint8_t* d_band_ok, int64_t t, int32_t* d_cand_idx, int32_t* d_act_slots,
                  int32_t* d_act_pix, int32_t* d_npos, void* stream);

/* Pre-load n forced positions (monitored for ever, BASELINE.json config 5) into the lowest free
 * slots; d_slots_out [n] (may be NULL).  Synchronises.  Returns LPF_E_STATE if the table is full and LPF_E_ARG if a
 * position lies outside the image (checked on the device; nothing is added in either case). */
int lpf_add_candidates(lpf_ctx* ctx, const int32_t* d_pix, int32_t n, int32_t* d_slots_out, void* stream);

/* -- S11: forced peak flux (O9) --------------------------------
 * d_flux [npos][B] = max of the raw cube over the (2 r_flux+1)^2 box, valid in-image pixels;
 * rejected band or frame -> 0.  d_pos is any pixel list (normally d_act_pix). */
int lpf_measure_flux(lpf_ctx* ctx, const float* d_cube, const uint8_t* d_band_ok, const int32_t* d_pos,
                     const int32_t* d_npos, float* d_flux, void* stream);

/* -- S12: ring append (O10) ------------------------------------
 * ring[slot][t mod T_ring][b] = flux; a slot born at t is pre-filled with NaN first. */
int lpf_append_dynspec(lpf_ctx* ctx, const int32_t* d_slots, const int32_t* d_n, const float* d_flux,
                       const uint8_t* d_band_ok, int64_t t, void* stream);

/* d_out [B][T_ring], time ordered oldest -> newest, ending at t_last (frequency x time, Fig. 1). */
int lpf_get_dynspec(lpf_ctx* ctx, int32_t slot, int64_t t_last, float* d_out, void* stream);

/* -- what the parameter-inference network is fed with ------------------------
 * d_out [n][B][T_ring] float32: the time-ordered dynamic spectra (as lpf_get_dynspec) of the n slots in d_slots,
 * each band divided by d_sigma[b] (its noise sigma, e.g. column 2 or 5 of the QC statistics; NULL or <= 0: 1),
 * samples that do not exist (before birth, outside the ring) set to 0 instead of NaN.  A batch (N, 1, B, T). */
int lpf_export_dynspec(lpf_ctx* ctx, const int32_t* d_slots, int32_t n, int64_t t_last, const float* d_sigma,
                       float* d_out, void* stream);
/* Simulated dispersed pulses, eqs. 19-21: for sample i with d_theta[i] = (t0 [steps], w [steps],
 * DM [pc/cm^3], A, alpha):  t_nu = t0 + 4148.806 s MHz^2 DM (nu^-2 - nu0^-2) / dt_s;
 * I(t, nu) = A (nu/nu0)^alpha exp[-1/2 ((t - t_nu)/w)^2]  (eq. 19 with the 1/2 its own FWHM implies, R18).
 * d_out [n][B][T] is overwritten (accumulate = 0) or added to (accumulate != 0: injection into noise or into
 * exported dynamic spectra).  d_nu [B] in MHz.  No context needed. */
int lpf_simulate_pulses(int32_t n, int32_t B, int32_t T, const float* d_nu, float nu0, float dt_s, const float* d_theta,
                        float* d_out, int32_t accumulate, void* stream);

/* -- whole step --------------------------------------------------------------
 * qc -> detect -> associate -> flux -> append for one cube on one lane, results in lane-owned
 * buffers (lpf_frame_view).  Frames on different lanes / streams overlap.  Contract: issue the calls in increasing t;
 * one stream per lane (a lane's buffers are reused by its next frame in stream order); with n_lanes lanes use them
 * round robin (the backward-fill cache holds n_back + n_lanes cubes: a lane that runs more than n_lanes frames ahead
 * of another would overwrite a cube that a frame in flight still needs).  Across lanes the context orders two
 * things itself: the association steps (all frames, in frame order, on a stream of its own) and the ring steps (an
 * event).  On the fused path with an aligned cube, no eq. A.2 and no backward fill, the lane's kernels are launched
 * as two CUDA graphs built at the lane's first frame; d_cube and t may change freely from call to call.
 * lpf_add_candidates synchronises the device (the table is shared with every frame in flight). */
int lpf_process_frame(lpf_ctx* ctx, int lane, const float* d_cube, int64_t t, void* stream);
int lpf_get_frame_view(lpf_ctx* ctx, int lane, lpf_frame_view* out);

/* Same step from HOST memory: copies h_cube (pinned for full speed) to the lane's device cube
 * buffer, runs the chain, copies the results back into `res`.  Synchronises `stream`. */
int lpf_process_frame_host(lpf_ctx* ctx, int lane, const float* h_cube, int64_t t, lpf_host_result* res,
                           void* stream);
/* The same call in two halves, so that several lanes can be in flight from the host: _begin enqueues the
 * copy in, the chain and the copy out of the counts / statistics on `stream` and returns at once
 * (h_cube and res must stay untouched until _end); _end waits for the stream, copies the variable-length
 * lists (nu, npos known by then) and returns with `res` filled (LPF_W_CAPACITY when the frame found more records
 * than max_det or more entries than cap_u / cap_pos hold: the lists are truncated).  One _begin per lane at a time;
 * issue the _begin calls in increasing t. */
int lpf_process_frame_host_begin(lpf_ctx* ctx, int lane, const float* h_cube, int64_t t, lpf_host_result* res,
                                 void* stream);
int lpf_process_frame_host_end(lpf_ctx* ctx, int lane, lpf_host_result* res, void* stream);

/* h_out[0] = records dropped (max_det; the fused path's hit list), h_out[1] = detections dropped (n_cand_max full),
 * h_out[2] = kernels launched by this context so far, h_out[3] = active candidates.  Synchronises.  Returns
 * LPF_W_CAPACITY when something was dropped since lpf_create (capacity overflow is never undefined behaviour:
 * the list is truncated and the drop counted). */
int lpf_get_counters(lpf_ctx* ctx, int64_t* h_out);

/* -- checkpoint / resume (optional; the method is a stream processor) ----------
 * Everything a context carries from one frame to the next, as one opaque blob in HOST memory: the candidate table
 * (PAPER.md:108), the dynamic-spectrum rings with their slot metadata, the drop counters, the running per-pixel state
 * of eq. A.2 and the backward-fill cache of recent cubes.  lpf_state_bytes: size of the blob for this context.
 * lpf_export_state: synchronises the device, then copies; `bytes` must be >= lpf_state_bytes.  lpf_import_state:
 * synchronises, checks that the blob was written by a context with identical lpf_params and image size
 * (LPF_E_ARG otherwise, nothing is changed), then overwrites the state: the next frame continues the exported
 * stream bit for bit.  The caller owns the buffer. */
int64_t lpf_state_bytes(const lpf_ctx* ctx);
int lpf_export_state(lpf_ctx* ctx, void* h_buf, int64_t bytes);
int lpf_import_state(lpf_ctx* ctx, const void* h_buf, int64_t bytes);

/* Launch plan chosen at lpf_create: h_out[0] = 1 if the fused single-pass detection kernel is in use
 * (box K = 12, k_mf = 3, n_iter = 1, Dx % 4 == 0; otherwise the general multi-kernel path),
 * [1] strip width in columns, [2] threads per CTA, [3] CTAs per plane, [4] dynamic shared memory
 * bytes per CTA, [5] planes, [6] SMs, [7] QC blocks per band.  lpf_params.force_general = 1 selects the
 * general path (used by the parity tests). */
int lpf_get_plan(lpf_ctx* ctx, int64_t* h_out);

/* Optional per-kernel timing with CUDA events recorded on the launching stream, around every kernel
 * this context launches between lpf_profile_begin and lpf_profile_end (both synchronise).
 * h_count[k] / h_ms[k]: launches and summed milliseconds of kernel id k, n >= lpf_profile_kernel_count().
 * Used by bench.py for the roofline of the dominant kernel; off by default (no events recorded). */
int lpf_profile_begin(lpf_ctx* ctx);
int lpf_profile_end(lpf_ctx* ctx, int32_t* h_count, float* h_ms, int32_t n);
/* The raw records of the profile in launch order, instead of the per-kernel sums: kernel id, start and end in
 * milliseconds after the first record's start (a timeline; with several lanes in flight the records overlap).
 * Ends the profile like lpf_profile_end.  Returns the number of records written (<= n_max), or a negative status. */
int lpf_profile_timeline(lpf_ctx* ctx, int32_t* h_kid, float* h_t0_ms, float* h_t1_ms, int32_t n_max);
int lpf_profile_kernel_count(void);
const char* lpf_profile_kernel_name(int kid);

/* Convenience for bindings: synchronous copy of `bytes` from device to host memory. */
int lpf_memcpy_d2h(void* h_dst, const void* d_src, int64_t bytes);

const char* lpf_strerror(int code);
const char* lpf_last_cuda_error(void);
int lpf_version(void);

#ifdef __cplusplus
}
#endif
#endif /* LPF_H_ */
