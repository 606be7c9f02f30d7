"""Thin Python binding of the C-ABI in include/lpf.h (argument marshalling only).

Every step of the path runs in the CUDA library ``liblpf_b200.so``; PyTorch is used
for device memory and streams only.  There is no CPU fallback: if the library is
missing or no CUDA device is present the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "liblpf_b200.so")
_lib = None

STATS_PER_BAND = 8


class LpfParams(C.Structure):
    _fields_ = [
        ("B", C.c_int32), ("Dy", C.c_int32), ("Dx", C.c_int32),
        ("kappa", C.c_float), ("k_max", C.c_int32), ("eps_rel", C.c_float),
        ("sigma_mf", C.c_float), ("k_mf", C.c_int32),
        ("bg_kernel", C.c_int32), ("s_bg", C.c_float), ("k_bg", C.c_int32),
        ("n_iter", C.c_int32), ("detect_sum_plane", C.c_int32),
        ("qc_tau", C.c_float), ("qc_clip", C.c_float),
        ("r_flux", C.c_int32), ("r_dedupe", C.c_int32), ("r_assoc", C.c_int32), ("n_forget", C.c_int32),
        ("T_ring", C.c_int32), ("n_cand_max", C.c_int32), ("max_det", C.c_int32), ("n_lanes", C.c_int32),
        ("n_back", C.c_int32),
        ("zeta_thr", C.c_float), ("zeta_nmax", C.c_int32), ("zeta_window", C.c_int32), ("zeta_warm", C.c_int32),
        ("zeta_reset", C.c_int32), ("force_general", C.c_int32),
    ]


class LpfFrameView(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in (
        "d_stats", "d_band_ok", "d_dets", "d_ndets", "d_upos", "d_uplane", "d_usnr", "d_nu", "d_cand_idx",
        "d_act_slots", "d_act_pix", "d_npos", "d_flux", "d_zeta_cnt")]


class LpfHostResult(C.Structure):
    _fields_ = [
        ("h_stats", C.c_void_p), ("h_band_ok", C.c_void_p), ("h_upos", C.c_void_p), ("h_uplane", C.c_void_p),
        ("h_usnr", C.c_void_p), ("h_cand_idx", C.c_void_p), ("cap_u", C.c_int32),
        ("h_act_slots", C.c_void_p), ("h_flux", C.c_void_p), ("cap_pos", C.c_int32),
        ("nu", C.c_int32), ("npos", C.c_int32), ("ndets", C.c_int32),
    ]


DET_DTYPE = np.dtype([("pix", "<i4"), ("plane", "<i2"), ("iter", "<i2"), ("f", "<f4"), ("c", "<f4"),
                      ("s", "<f4"), ("snr", "<f4")])

EXPORTS = [
    "lpf_create", "lpf_destroy", "lpf_cube_qc", "lpf_detect_sources", "lpf_associate", "lpf_add_candidates",
    "lpf_measure_flux", "lpf_append_dynspec", "lpf_get_dynspec", "lpf_process_frame", "lpf_get_frame_view",
    "lpf_process_frame_host", "lpf_process_frame_host_begin", "lpf_process_frame_host_end", "lpf_get_counters", "lpf_memcpy_d2h", "lpf_strerror", "lpf_last_cuda_error",
    "lpf_export_dynspec", "lpf_simulate_pulses", "lpf_state_bytes", "lpf_export_state", "lpf_import_state", "lpf_cube_qc_static",
    "lpf_version", "lpf_get_plan", "lpf_profile_begin", "lpf_profile_end", "lpf_profile_timeline", "lpf_profile_kernel_count", "lpf_profile_kernel_name",
]


class LpfError(RuntimeError):
    pass


def load_library(path: Optional[str] = None):
    """dlopen the CUDA library; fails loudly if it has not been built."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    path = path or LIB_PATH
    if not os.path.exists(path):
        raise LpfError(f"{path} not found: build it with `python -m paper_2103_15418_b200.build` "
                       "(there is no CPU fallback)")
    lib = C.CDLL(path)
    vp, i32, i64 = C.c_void_p, C.c_int32, C.c_int64
    lib.lpf_create.argtypes = [C.POINTER(vp), C.POINTER(LpfParams), vp]
    lib.lpf_destroy.argtypes = [vp]
    lib.lpf_cube_qc.argtypes = [vp, C.c_int, vp, i64, vp, vp, vp]
    lib.lpf_detect_sources.argtypes = [vp, C.c_int, vp, vp, vp, vp, vp, vp, vp, vp, vp]
    lib.lpf_associate.argtypes = [vp, C.c_int, vp, vp, vp, i64, vp, vp, vp, vp, vp]
    lib.lpf_add_candidates.argtypes = [vp, vp, i32, vp, vp]
    lib.lpf_measure_flux.argtypes = [vp, vp, vp, vp, vp, vp, vp]
    lib.lpf_append_dynspec.argtypes = [vp, vp, vp, vp, vp, i64, vp]
    lib.lpf_get_dynspec.argtypes = [vp, i32, i64, vp, vp]
    lib.lpf_export_dynspec.argtypes = [vp, vp, i32, i64, vp, vp, vp]
    lib.lpf_simulate_pulses.argtypes = [i32, i32, i32, vp, C.c_float, C.c_float, vp, vp, i32, vp]
    lib.lpf_process_frame.argtypes = [vp, C.c_int, vp, i64, vp]
    lib.lpf_get_frame_view.argtypes = [vp, C.c_int, C.POINTER(LpfFrameView)]
    lib.lpf_process_frame_host.argtypes = [vp, C.c_int, vp, i64, C.POINTER(LpfHostResult), vp]
    lib.lpf_process_frame_host_begin.argtypes = [vp, C.c_int, vp, i64, C.POINTER(LpfHostResult), vp]
    lib.lpf_process_frame_host_end.argtypes = [vp, C.c_int, C.POINTER(LpfHostResult), vp]
    lib.lpf_get_counters.argtypes = [vp, C.POINTER(i64)]
    lib.lpf_memcpy_d2h.argtypes = [vp, vp, i64]
    lib.lpf_cube_qc_static.argtypes = [vp, vp, vp, vp, vp]
    lib.lpf_state_bytes.argtypes = [vp]
    lib.lpf_export_state.argtypes = [vp, vp, i64]
    lib.lpf_import_state.argtypes = [vp, vp, i64]
    lib.lpf_strerror.argtypes = [C.c_int]
    lib.lpf_strerror.restype = C.c_char_p
    lib.lpf_last_cuda_error.restype = C.c_char_p
    lib.lpf_get_plan.argtypes = [vp, C.POINTER(i64)]
    lib.lpf_profile_begin.argtypes = [vp]
    lib.lpf_profile_end.argtypes = [vp, vp, vp, i32]
    lib.lpf_profile_timeline.argtypes = [vp, vp, vp, vp, i32]
    lib.lpf_profile_kernel_name.argtypes = [C.c_int]
    lib.lpf_profile_kernel_name.restype = C.c_char_p
    for n in EXPORTS:
        if n not in ("lpf_strerror", "lpf_last_cuda_error", "lpf_profile_kernel_name", "lpf_state_bytes"):
            getattr(lib, n).restype = C.c_int
    lib.lpf_state_bytes.restype = i64
    if path == LIB_PATH:
        _lib = lib
    return lib


E_TOO_LARGE = -5   # the problem exceeds a fixed maximum of the entry point (include/lpf.h)
W_CAPACITY = 1   # positive status = warning: a list was truncated, the call did its work (include/lpf.h)


def _check(lib, rc: int, what: str):
    """Negative status: raise.  Positive (LPF_W_CAPACITY): a warning, returned to the caller."""
    if rc < 0:
        raise LpfError(f"{what}: {lib.lpf_strerror(rc).decode()} ({rc}) {lib.lpf_last_cuda_error().decode()}")


def make_params(p: dict) -> LpfParams:
    s = LpfParams()
    for name, _ in LpfParams._fields_:
        setattr(s, name, p[name] if name not in ("zeta_reset", "force_general") else p.get(name, 0))
    return s


def _ptr(t) -> int:
    return 0 if t is None else t.data_ptr()


def _stream(stream) -> int:
    import torch
    if stream is None:
        return torch.cuda.current_stream().cuda_stream
    return stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream)


class LPF:
    """One context (``lpf_ctx``).  Methods mirror the C-ABI names without the ``lpf_`` prefix and take
    torch CUDA tensors; they allocate outputs when none are passed."""

    def __init__(self, params: dict, mask=None, device: str = "cuda:0"):
        import torch
        if not torch.cuda.is_available():
            raise LpfError("no CUDA device: the LPF path has no CPU fallback")
        self.torch = torch
        self.lib = load_library()
        self.p = dict(params)
        self.dev = torch.device(device)
        torch.cuda.set_device(self.dev)
        self.B, self.Dy, self.Dx = self.p["B"], self.p["Dy"], self.p["Dx"]
        self._mask = None
        if mask is not None:
            self._mask = torch.as_tensor(np.ascontiguousarray(mask, dtype=np.uint8)).to(self.dev)
        h = C.c_void_p()
        sp = make_params(self.p)
        _check(self.lib, self.lib.lpf_create(C.byref(h), C.byref(sp), _ptr(self._mask)), "lpf_create")
        self.h = h

    def close(self):
        if getattr(self, "h", None):
            self.lib.lpf_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- allocation helpers ---------------------------------------------------
    def _empty(self, shape, dtype):
        return self.torch.empty(shape, dtype=dtype, device=self.dev)

    # -- C-ABI mirrors ----------------------------------------------------------
    def cube_qc(self, cube, t: int = 0, lane: int = 0, stream=None):
        tc = self.torch
        stats = self._empty((self.B, STATS_PER_BAND), tc.float32)
        ok = self._empty((self.B + 1,), tc.uint8)
        _check(self.lib, self.lib.lpf_cube_qc(self.h, lane, _ptr(cube), t, _ptr(stats), _ptr(ok), _stream(stream)), "lpf_cube_qc")
        return stats, ok

    def cube_qc_static(self, cube, stats=None, ok=None, stream=None):
        """lpf_cube_qc_static: the statistics and eq. A.1 verdict with their scratch in the library's static device
        array; the call allocates nothing when the caller passes `stats` [B][8] float32 and `ok` [B + 1] uint8."""
        tc = self.torch
        if stats is None:
            stats = self._empty((self.B, STATS_PER_BAND), tc.float32)
        if ok is None:
            ok = self._empty((self.B + 1,), tc.uint8)
        _check(self.lib, self.lib.lpf_cube_qc_static(self.h, _ptr(cube), _ptr(stats), _ptr(ok), _stream(stream)), "lpf_cube_qc_static")
        return stats, ok

    def detect_sources(self, cube, band_ok, lane: int = 0, stream=None):
        tc = self.torch
        md = self.p["max_det"]
        dets = self._empty((md * DET_DTYPE.itemsize,), tc.uint8)
        ndets = self._empty((1,), tc.int32)
        upos = self._empty((md,), tc.int32); uplane = self._empty((md,), tc.int16); usnr = self._empty((md,), tc.float32)
        nu = self._empty((1,), tc.int32)
        _check(self.lib, self.lib.lpf_detect_sources(self.h, lane, _ptr(cube), _ptr(band_ok), _ptr(dets), _ptr(ndets),
                                                     _ptr(upos), _ptr(uplane), _ptr(usnr), _ptr(nu), _stream(stream)),
               "lpf_detect_sources")
        return dict(dets=dets, ndets=ndets, upos=upos, uplane=uplane, usnr=usnr, nu=nu)

    def associate(self, upos, nu, band_ok, t: int, lane: int = 0, stream=None):
        tc = self.torch
        cand = self._empty((max(int(upos.numel()), 1),), tc.int32)
        act_s = self._empty((self.p["n_cand_max"],), tc.int32); act_p = self._empty((self.p["n_cand_max"],), tc.int32)
        npos = self._empty((1,), tc.int32)
        _check(self.lib, self.lib.lpf_associate(self.h, lane, _ptr(upos), _ptr(nu), _ptr(band_ok), t, _ptr(cand),
                                                _ptr(act_s), _ptr(act_p), _ptr(npos), _stream(stream)), "lpf_associate")
        return dict(cand_idx=cand, act_slots=act_s, act_pix=act_p, npos=npos)

    def add_candidates(self, pix, stream=None):
        tc = self.torch
        pix = tc.as_tensor(np.ascontiguousarray(pix, dtype=np.int32)).to(self.dev) if not tc.is_tensor(pix) else pix
        out = self._empty((max(int(pix.numel()), 1),), tc.int32)
        _check(self.lib, self.lib.lpf_add_candidates(self.h, _ptr(pix), int(pix.numel()), _ptr(out), _stream(stream)),
               "lpf_add_candidates")
        return out[:pix.numel()]

    def measure_flux(self, cube, band_ok, pos, npos, stream=None):
        flux = self._empty((max(int(pos.numel()), 1), self.B), self.torch.float32)
        _check(self.lib, self.lib.lpf_measure_flux(self.h, _ptr(cube), _ptr(band_ok), _ptr(pos), _ptr(npos), _ptr(flux),
                                                   _stream(stream)), "lpf_measure_flux")
        return flux

    def append_dynspec(self, slots, n, flux, band_ok, t: int, stream=None):
        _check(self.lib, self.lib.lpf_append_dynspec(self.h, _ptr(slots), _ptr(n), _ptr(flux), _ptr(band_ok), t,
                                                     _stream(stream)), "lpf_append_dynspec")

    def get_dynspec(self, slot: int, t_last: int, stream=None):
        out = self._empty((self.B, self.p["T_ring"]), self.torch.float32)
        _check(self.lib, self.lib.lpf_get_dynspec(self.h, int(slot), int(t_last), _ptr(out), _stream(stream)), "lpf_get_dynspec")
        return out

    def process_frame(self, cube, t: int, lane: int = 0, stream=None):
        _check(self.lib, self.lib.lpf_process_frame(self.h, lane, _ptr(cube), t, _stream(stream)), "lpf_process_frame")

    def frame_view(self, lane: int = 0) -> dict:
        """Copy a lane's results to host numpy arrays (synchronises)."""
        import torch
        v = LpfFrameView()
        _check(self.lib, self.lib.lpf_get_frame_view(self.h, lane, C.byref(v)), "lpf_get_frame_view")
        torch.cuda.synchronize()

        def rd(ptr, n, dtype):
            out = np.empty(n, dtype=dtype)
            if n:
                _check(self.lib, self.lib.lpf_memcpy_d2h(out.ctypes.data, ptr, out.nbytes), "lpf_memcpy_d2h")
            return out
        B = self.B
        nu = int(rd(v.d_nu, 1, np.int32)[0]); npos = int(rd(v.d_npos, 1, np.int32)[0])
        ndets = int(rd(v.d_ndets, 1, np.int32)[0])
        nd = min(ndets, self.p["max_det"])
        return dict(
            stats=rd(v.d_stats, B * STATS_PER_BAND, np.float32).reshape(B, STATS_PER_BAND),
            band_ok=rd(v.d_band_ok, B + 1, np.uint8),
            rec=rd(v.d_dets, nd, DET_DTYPE), ndets=ndets,
            upos=rd(v.d_upos, nu, np.int32), uplane=rd(v.d_uplane, nu, np.int16), usnr=rd(v.d_usnr, nu, np.float32),
            cand_idx=rd(v.d_cand_idx, nu, np.int32),
            act_slots=rd(v.d_act_slots, npos, np.int32), act_pix=rd(v.d_act_pix, npos, np.int32),
            flux=rd(v.d_flux, npos * B, np.float32).reshape(npos, B),
            zeta_cnt=rd(v.d_zeta_cnt, B, np.int32),
        )

    def process_frame_host(self, h_cube, t: int, res: "HostResult", lane: int = 0, stream=None):
        """h_cube: pinned CPU torch tensor (or numpy array) [B,Dy,Dx] float32."""
        ptr = h_cube.data_ptr() if hasattr(h_cube, "data_ptr") else h_cube.ctypes.data
        _check(self.lib, self.lib.lpf_process_frame_host(self.h, lane, ptr, t, C.byref(res.c), _stream(stream)),
               "lpf_process_frame_host")
        return res

    def process_frame_host_begin(self, h_cube, t: int, res: "HostResult", lane: int = 0, stream=None):
        ptr = h_cube.data_ptr() if hasattr(h_cube, "data_ptr") else h_cube.ctypes.data
        _check(self.lib, self.lib.lpf_process_frame_host_begin(self.h, lane, ptr, t, C.byref(res.c), _stream(stream)),
               "lpf_process_frame_host_begin")

    def process_frame_host_end(self, res: "HostResult", lane: int = 0, stream=None):
        rc = self.lib.lpf_process_frame_host_end(self.h, lane, C.byref(res.c), _stream(stream))
        _check(self.lib, rc, "lpf_process_frame_host_end")
        res.truncated = rc == W_CAPACITY
        return res

    def export_dynspec(self, slots, t_last: int, sigma=None, stream=None):
        """[n][B][T_ring] float32 network input: ordered, sigma-normalised, NaN-free dynamic spectra."""
        import torch
        n = int(slots.numel())
        out = torch.empty((n, self.B, self.p["T_ring"]), dtype=torch.float32, device=slots.device)
        _check(self.lib, self.lib.lpf_export_dynspec(self.h, _ptr(slots), n, t_last, _ptr(sigma), _ptr(out), _stream(stream)),
               "lpf_export_dynspec")
        return out

    def plan(self) -> dict:
        h = (C.c_int64 * 8)()
        _check(self.lib, self.lib.lpf_get_plan(self.h, h), "lpf_get_plan")
        return dict(fused=bool(h[0]), strip_cols=int(h[1]), threads=int(h[2]), ctas_per_plane=int(h[3]),
                    smem_bytes=int(h[4]), planes=int(h[5]), sms=int(h[6]), qc_blocks_per_band=int(h[7]))

    def profile_begin(self):
        _check(self.lib, self.lib.lpf_profile_begin(self.h), "lpf_profile_begin")

    def profile_end(self) -> dict:
        """{kernel name: (launches, total ms)} for every kernel launched since profile_begin."""
        n = self.lib.lpf_profile_kernel_count()
        cnt = (C.c_int32 * n)(); ms = (C.c_float * n)()
        _check(self.lib, self.lib.lpf_profile_end(self.h, cnt, ms, n), "lpf_profile_end")
        return {self.lib.lpf_profile_kernel_name(i).decode(): (int(cnt[i]), float(ms[i])) for i in range(n) if cnt[i]}

    def profile_timeline(self, n_max: int = 65536):
        """[(kernel name, start ms, end ms)] of every kernel launched since profile_begin, in launch order."""
        kid = (C.c_int32 * n_max)(); t0 = (C.c_float * n_max)(); t1 = (C.c_float * n_max)()
        n = self.lib.lpf_profile_timeline(self.h, kid, t0, t1, n_max)
        if n < 0:
            _check(self.lib, n, "lpf_profile_timeline")
        return [(self.lib.lpf_profile_kernel_name(kid[i]).decode(), float(t0[i]), float(t1[i])) for i in range(n)]

    def export_state(self) -> np.ndarray:
        """Everything the context carries from frame to frame, as one host blob (lpf_export_state)."""
        n = int(self.lib.lpf_state_bytes(self.h))
        if n < 0:
            _check(self.lib, n, "lpf_state_bytes")
        buf = np.empty(n, np.uint8)
        _check(self.lib, self.lib.lpf_export_state(self.h, buf.ctypes.data, n), "lpf_export_state")
        return buf

    def import_state(self, buf: np.ndarray) -> None:
        buf = np.ascontiguousarray(buf, dtype=np.uint8)
        _check(self.lib, self.lib.lpf_import_state(self.h, buf.ctypes.data, buf.nbytes), "lpf_import_state")

    def counters(self) -> dict:
        h = (C.c_int64 * 4)()
        rc = self.lib.lpf_get_counters(self.h, h)
        _check(self.lib, rc, "lpf_get_counters")
        return dict(dropped_records=int(h[0]), dropped_detections=int(h[1]), launches=int(h[2]), n_active=int(h[3]),
                    truncated=rc == W_CAPACITY)


class HostResult:
    """Pinned host buffers for ``lpf_process_frame_host``."""

    def __init__(self, params: dict, cap_u: int = 65536, cap_pos: Optional[int] = None):
        import torch
        B = params["B"]
        cap_pos = cap_pos or params["n_cand_max"]
        pin = dict(pin_memory=True)
        self.stats = torch.empty((B, STATS_PER_BAND), dtype=torch.float32, **pin)
        self.band_ok = torch.empty((B + 1,), dtype=torch.uint8, **pin)
        self.upos = torch.empty((cap_u,), dtype=torch.int32, **pin)
        self.uplane = torch.empty((cap_u,), dtype=torch.int16, **pin)
        self.usnr = torch.empty((cap_u,), dtype=torch.float32, **pin)
        self.cand_idx = torch.empty((cap_u,), dtype=torch.int32, **pin)
        self.act_slots = torch.empty((cap_pos,), dtype=torch.int32, **pin)
        self.flux = torch.empty((cap_pos, B), dtype=torch.float32, **pin)
        c = LpfHostResult()
        c.h_stats = self.stats.data_ptr(); c.h_band_ok = self.band_ok.data_ptr()
        c.h_upos = self.upos.data_ptr(); c.h_uplane = self.uplane.data_ptr(); c.h_usnr = self.usnr.data_ptr()
        c.h_cand_idx = self.cand_idx.data_ptr(); c.cap_u = cap_u
        c.h_act_slots = self.act_slots.data_ptr(); c.h_flux = self.flux.data_ptr(); c.cap_pos = cap_pos
        self.c = c

    @property
    def nu(self):
        return int(self.c.nu)

    @property
    def npos(self):
        return int(self.c.npos)

    @property
    def d2h_bytes(self):
        B = self.stats.shape[0]
        return B * STATS_PER_BAND * 4 + B + 1 + 12 + self.nu * 14 + self.npos * (4 + 4 * B)


def simulate_pulses(theta, nu, nu0: float, T: int, dt_s: float = 1.0, out=None, accumulate: bool = False, stream=None):
    """Simulated dispersed pulses (eqs. 19-21): theta [n][5] = (t0, w, DM, A, alpha), nu [B] MHz -> [n][B][T] (CUDA tensors)."""
    import torch
    lib = load_library()
    n, B = int(theta.shape[0]), int(nu.numel())
    if out is None:
        out = torch.empty((n, B, T), dtype=torch.float32, device=theta.device)
        accumulate = False
    _check(lib, lib.lpf_simulate_pulses(n, B, T, _ptr(nu), float(nu0), float(dt_s), _ptr(theta), _ptr(out), int(bool(accumulate)),
                                        _stream(stream)), "lpf_simulate_pulses")
    return out
