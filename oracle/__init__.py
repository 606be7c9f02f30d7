"""CPU oracle for the LPF hot path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

A ctypes wrapper around ``oracle/lpf_oracle.cpp`` (plain single-threaded float64
C++ written from the paper) plus :class:`OraclePipeline`, which chains the steps in
the paper's order (Fig. 2 :35, Fig. 4 :116).

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It imports nothing from the
CUDA package (``paper_2103_15418_b200``) and shares no code with it.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lpf_oracle.cpp")
_LIB = os.path.join(_HERE, "liblpf_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (no OpenMP, no -ffast-math)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-Wno-stringop-overflow", "-fPIC", "-shared", "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_LIB)
        _lib.orc_associate.restype = C.c_int
        _lib.orc_dedupe.restype = C.c_int
        _lib.orc_version.restype = C.c_int
    return _lib


def _p(a, t):
    return None if a is None else a.ctypes.data_as(C.POINTER(t))


def _mask_arg(W):
    if W is None:
        return None, None
    W = np.ascontiguousarray(W, dtype=np.uint8)
    return W, _p(W, C.c_uint8)


# ----------------------------------------------------------------------------
def band_stats(cube: np.ndarray, W: Optional[np.ndarray], qc_clip: float) -> np.ndarray:
    """O1 -> [B][6] = n, mean, rms, n_clip, clipped mean, clipped rms (float64)."""
    cube = np.ascontiguousarray(cube, dtype=np.float32)
    B, Dy, Dx = cube.shape
    Wk, Wp = _mask_arg(W)
    out = np.zeros((B, 6), dtype=np.float64)
    lib().orc_band_stats(_p(cube, C.c_float), B, Dy, Dx, Wp, C.c_double(qc_clip), _p(out, C.c_double))
    return out


def qc_verdict(stats: np.ndarray, tau: float):
    """O2 -> (z [B][2], band_ok uint8 [B+1] with band_ok[B] = frame_ok)."""
    stats = np.ascontiguousarray(stats, dtype=np.float64)
    B = stats.shape[0]
    z = np.zeros((B, 2), dtype=np.float64)
    ok = np.zeros(B + 1, dtype=np.uint8)
    lib().orc_qc_verdict(_p(stats, C.c_double), B, C.c_double(tau), _p(z, C.c_double), _p(ok, C.c_uint8))
    return z, ok


def kernel_taps(kind: int, s: float, k: int) -> np.ndarray:
    """O3.  kind 0 = Gaussian (eq. 2), 1 = uniform; s <= 0 (kind 0) = identity."""
    g = np.zeros(2 * k + 1, dtype=np.float64)
    lib().orc_kernel_taps(int(kind), C.c_double(s), int(k), _p(g, C.c_double))
    return g


def normconv(A: np.ndarray, Wp: Optional[np.ndarray], g: np.ndarray, direct: bool = True, want_den: bool = False):
    A = np.ascontiguousarray(A, dtype=np.float64)
    Dy, Dx = A.shape
    g = np.ascontiguousarray(g, dtype=np.float64)
    k = (g.size - 1) // 2
    Wk, Wptr = _mask_arg(Wp)
    out = np.zeros_like(A)
    den = np.zeros_like(A) if want_den else None
    lib().orc_normconv(_p(A, C.c_double), Wptr, Dy, Dx, _p(g, C.c_double), k, int(bool(direct)),
                       _p(out, C.c_double), _p(den, C.c_double))
    return (out, den) if want_den else out


def planes(cube: np.ndarray, band_ok: np.ndarray) -> np.ndarray:
    """O4 -> [B+1][Dy][Dx] float64; plane B = sum of accepted bands."""
    cube = np.ascontiguousarray(cube, dtype=np.float32)
    B, Dy, Dx = cube.shape
    band_ok = np.ascontiguousarray(band_ok, dtype=np.uint8)
    out = np.zeros((B + 1, Dy, Dx), dtype=np.float64)
    lib().orc_planes(_p(cube, C.c_float), _p(band_ok, C.c_uint8), B, Dy, Dx, _p(out, C.c_double))
    return out


def detect_plane(X: np.ndarray, W: Optional[np.ndarray], params: dict, direct: bool = True) -> dict:
    """O4-O6 for one plane.  Returns dict(F, iter, C, S, snr, Q, P, C_last, S_last)."""
    X = np.ascontiguousarray(X, dtype=np.float64)
    Dy, Dx = X.shape
    Wk, Wptr = _mask_arg(W)
    g_mf = kernel_taps(0, params["sigma_mf"], params["k_mf"])
    g_bg = kernel_taps(params["bg_kernel"], params["s_bg"], params["k_bg"])
    F = np.zeros((Dy, Dx)); Cd = np.zeros((Dy, Dx)); Sd = np.zeros((Dy, Dx)); snr = np.zeros((Dy, Dx))
    Cl = np.zeros((Dy, Dx)); Sl = np.zeros((Dy, Dx))
    it = np.zeros((Dy, Dx), dtype=np.uint8); Q = np.zeros((Dy, Dx), dtype=np.uint8); P = np.zeros((Dy, Dx), dtype=np.uint8)
    lib().orc_detect_plane(_p(X, C.c_double), Wptr, Dy, Dx,
                           _p(g_mf, C.c_double), int(params["k_mf"]), _p(g_bg, C.c_double), int(params["k_bg"]),
                           C.c_double(params["kappa"]), C.c_double(params["eps_rel"]), int(params["n_iter"]),
                           int(params["k_max"]), int(bool(direct)),
                           _p(F, C.c_double), _p(it, C.c_uint8), _p(Cd, C.c_double), _p(Sd, C.c_double),
                           _p(snr, C.c_double), _p(Q, C.c_uint8), _p(P, C.c_uint8),
                           _p(Cl, C.c_double), _p(Sl, C.c_double))
    return dict(F=F, iter=it, C=Cd, S=Sd, snr=snr, Q=Q, P=P, C_last=Cl, S_last=Sl)


def dedupe(pix, plane, snr, Dy: int, Dx: int, r_dedupe: int):
    """O7 -> (upos int32, uplane int16, usnr float64), sorted by pix."""
    pix = np.ascontiguousarray(pix, dtype=np.int32)
    plane = np.ascontiguousarray(plane, dtype=np.int16)
    snr = np.ascontiguousarray(snr, dtype=np.float64)
    n = pix.size
    upos = np.zeros(max(n, 1), dtype=np.int32); upl = np.zeros(max(n, 1), dtype=np.int16); us = np.zeros(max(n, 1))
    nu = lib().orc_dedupe(_p(pix, C.c_int32), _p(plane, C.c_int16), _p(snr, C.c_double), n, Dy, Dx, int(r_dedupe),
                          _p(upos, C.c_int32), _p(upl, C.c_int16), _p(us, C.c_double))
    return upos[:nu].copy(), upl[:nu].copy(), us[:nu].copy()


def measure_flux(cube, band_ok, W, pos, r_flux: int) -> np.ndarray:
    """O9 -> [npos][B] float32."""
    cube = np.ascontiguousarray(cube, dtype=np.float32)
    B, Dy, Dx = cube.shape
    band_ok = np.ascontiguousarray(band_ok, dtype=np.uint8)
    pos = np.ascontiguousarray(pos, dtype=np.int32)
    Wk, Wptr = _mask_arg(W)
    out = np.zeros((pos.size, B), dtype=np.float32)
    lib().orc_measure_flux(_p(cube, C.c_float), _p(band_ok, C.c_uint8), Wptr, B, Dy, Dx,
                           _p(pos, C.c_int32), int(pos.size), int(r_flux), _p(out, C.c_float))
    return out


class RunningQC:
    """O12, per-pixel running quality control (eq. A.2; R22).

    State per band and pixel: running mean m and variance v of the image stream -- float32 IMAGES, like the
    cube itself (:389 "running mean and standard deviation images") -- and the number of updates n_b.
    Welford (1962) while the band has fewer than `window` updates, exponentially weighted after that
    (Finch 2009): one recurrence, a = 1/min(n_b + 1, window), d = x - m, m += a d, v = (1 - a)(v + a d^2).
    For a frame: zeta = (x - m)/sqrt(v) (eq. A.2) at every valid pixel with v > 0 of every band with
    n_b >= warm; the band is discarded when more than `nmax` pixels have |zeta| > thr (nmax = 0: the
    paper's "if zeta exceeds a threshold").  The test comes before the update, and only bands that survive
    both eq. A.1 and eq. A.2 update their state.  A band discarded by eq. A.2 in `reset` consecutive frames
    (reset > 0) starts over (n_b = 0: Welford from scratch, untested during the warm-up) -- the way out of a
    lasting level change.

    All arithmetic is float64 on the float32 state; each new state value is rounded to float32 once.
    |zeta| > thr is evaluated as d^2 > thr^2 v.  `near[b]` counts the valid pixels whose decision is within
    2e-4 relative of the threshold (the parity harness accepts a count difference only up to that number).
    """

    def __init__(self, B: int, Dy: int, Dx: int, thr: float, nmax: int, window: int, warm: int, reset: int = 0):
        self.thr2 = float(thr) ** 2; self.nmax = int(nmax)
        self.window = int(window); self.warm = int(warm); self.reset = int(reset)
        self.m = np.zeros((B, Dy, Dx), np.float32); self.v = np.zeros((B, Dy, Dx), np.float32)
        self.n = np.zeros(B, np.int32)
        self.run = np.zeros(B, np.int32)          # consecutive eq. A.2 discards
        self.near = np.zeros(B, np.int32)

    def step(self, cube, W, band_ok):
        """band_ok: [B+1] after eq. A.1.  Returns (counts [B] int32, band_ok' [B+1])."""
        cube = np.asarray(cube, np.float32)
        B = cube.shape[0]
        ok = np.array(band_ok, np.uint8, copy=True)
        cnt = np.zeros(B, np.int32)
        self.near[:] = 0
        valid = np.ones(cube.shape[1:], bool) if W is None else (np.asarray(W) != 0)
        for b in range(B):
            with np.errstate(invalid="ignore", over="ignore"):
                m = self.m[b].astype(np.float64); v = self.v[b].astype(np.float64)
                d = cube[b].astype(np.float64) - m
                a1_ok = bool(ok[b]); discard = False
                if self.n[b] >= self.warm:
                    lhs = d * d; rhs = self.thr2 * v
                    tested = valid & (v > 0)
                    cnt[b] = int(np.count_nonzero((lhs > rhs) & tested))
                    self.near[b] = int(np.count_nonzero((np.abs(lhs - rhs) <= 2e-4 * rhs) & tested))
                    discard = cnt[b] > self.nmax
                if discard:
                    ok[b] = 0
                if ok[b]:
                    a = 1.0 / min(int(self.n[b]) + 1, self.window)
                    self.m[b] = (m + a * d).astype(np.float32)
                    self.v[b] = ((1.0 - a) * (v + a * d * d)).astype(np.float32)
                    self.n[b] += 1
                    self.run[b] = 0
                elif a1_ok and discard:
                    self.run[b] += 1
                    if self.reset > 0 and self.run[b] >= self.reset:
                        self.m[b] = 0; self.v[b] = 0; self.n[b] = 0; self.run[b] = 0
        ok[B] = 1 if int(ok[:B].sum()) >= (B + 1) // 2 else 0
        return cnt, ok


class CandidateTable:
    """O8 + O10 state: candidate table and dynamic-spectrum rings."""

    def __init__(self, n_cand_max: int, T_ring: int, B: int, Dx: int, r_assoc: int, n_forget: int):
        self.n = n_cand_max; self.T = T_ring; self.B = B; self.Dx = Dx
        self.r_assoc = r_assoc; self.n_forget = n_forget
        self.active = np.zeros(n_cand_max, dtype=np.uint8)
        self.forced = np.zeros(n_cand_max, dtype=np.uint8)
        self.cpix = np.zeros(n_cand_max, dtype=np.int32)
        self.miss = np.zeros(n_cand_max, dtype=np.int32)
        self.born = np.full(n_cand_max, -1, dtype=np.int64)
        self.ring = np.full((n_cand_max, T_ring, B), np.nan, dtype=np.float32)
        self.meta_t = np.full(T_ring, -1, dtype=np.int64)
        self.meta_ok = np.zeros(T_ring, dtype=np.uint64)
        self.n_dropped = np.zeros(1, dtype=np.int32)
        self.t_last = -1

    def add_forced(self, pix) -> np.ndarray:
        """Pre-load forced positions (never retired) into the lowest free slots."""
        pix = np.asarray(pix, dtype=np.int32)
        free = np.flatnonzero(self.active == 0)[:pix.size]
        assert free.size == pix.size, "candidate table full"
        self.active[free] = 1; self.forced[free] = 1; self.cpix[free] = pix
        self.miss[free] = 0; self.born[free] = -1
        self.ring[free] = np.nan
        return free.astype(np.int32)

    def associate(self, upos, t: int, frame_ok: int):
        upos = np.ascontiguousarray(upos, dtype=np.int32)
        nu = upos.size
        cand = np.zeros(max(nu, 1), dtype=np.int32)
        act_s = np.zeros(self.n, dtype=np.int32); act_p = np.zeros(self.n, dtype=np.int32)
        na = lib().orc_associate(_p(self.active, C.c_uint8), _p(self.forced, C.c_uint8), _p(self.cpix, C.c_int32),
                                 _p(self.miss, C.c_int32), _p(self.born, C.c_int64), self.n,
                                 _p(upos, C.c_int32), nu, C.c_int64(t), int(frame_ok),
                                 self.Dx, self.r_assoc, self.n_forget,
                                 _p(cand, C.c_int32), _p(act_s, C.c_int32), _p(act_p, C.c_int32),
                                 _p(self.n_dropped, C.c_int32))
        return cand[:nu].copy(), act_s[:na].copy(), act_p[:na].copy()

    def append(self, slots, flux, band_ok, t: int):
        slots = np.ascontiguousarray(slots, dtype=np.int32)
        flux = np.ascontiguousarray(flux, dtype=np.float32)
        band_ok = np.ascontiguousarray(band_ok, dtype=np.uint8)
        lib().orc_ring_append(_p(self.ring, C.c_float), _p(self.meta_t, C.c_int64), _p(self.meta_ok, C.c_uint64),
                              _p(self.born, C.c_int64), self.T, self.B, _p(slots, C.c_int32), int(slots.size),
                              _p(flux, C.c_float), _p(band_ok, C.c_uint8), C.c_int64(t))
        self.t_last = t

    def dynspec(self, slot: int, t_last: Optional[int] = None) -> np.ndarray:
        out = np.zeros((self.B, self.T), dtype=np.float32)
        tl = self.t_last if t_last is None else t_last
        lib().orc_get_dynspec(_p(self.ring, C.c_float), _p(self.meta_t, C.c_int64), self.T, self.B, int(slot),
                              C.c_int64(tl), _p(out, C.c_float))
        return out


class OraclePipeline:
    """Whole per-time-step chain in the paper's order:
    QC -> planes -> per-plane detection -> dedupe -> associate -> flux -> ring."""

    def __init__(self, params: dict, mask: Optional[np.ndarray] = None, direct: bool = True):
        self.p = dict(params)
        self.W = None if mask is None else np.ascontiguousarray(mask, dtype=np.uint8)
        self.direct = direct
        p = self.p
        self.table = CandidateTable(p["n_cand_max"], p["T_ring"], p["B"], p["Dx"], p["r_assoc"], p["n_forget"])
        self.n_back = int(p.get("n_back", 0))
        self.rq = None
        if float(p.get("zeta_thr", 0.0)) > 0:
            self.rq = RunningQC(p["B"], p["Dy"], p["Dx"], p["zeta_thr"], p.get("zeta_nmax", 0), p.get("zeta_window", 64),
                                p.get("zeta_warm", 8), p.get("zeta_reset", 0))
        self.zeta_cnt = np.zeros(p["B"], np.int32)
        self.history = []   # O11: the last n_back frames as (t, cube, band_ok)

    # -- steps ---------------------------------------------------------------
    def cube_qc(self, cube):
        st = band_stats(cube, self.W, self.p["qc_clip"])
        z, ok = qc_verdict(st, self.p["qc_tau"])
        if self.rq is not None:                       # eq. A.2 after eq. A.1 (O12)
            self.zeta_cnt, ok = self.rq.step(cube, self.W, ok)
        return np.concatenate([st, z], axis=1), ok  # [B][8], [B+1]

    def detect(self, cube, band_ok, keep_planes: bool = False):
        p = self.p
        B = p["B"]
        recs = []  # (plane, pix, iter, f, c, s, snr)
        per_plane = []
        if band_ok[B]:
            pl = planes(cube, band_ok)
            n_planes = B + 1 if p.get("detect_sum_plane", 1) else B
            for q in range(n_planes):
                if q < B and not band_ok[q]:
                    per_plane.append(None)
                    continue
                d = detect_plane(pl[q], self.W, p, self.direct)
                pix = np.flatnonzero(d["P"].ravel())
                for i in pix:
                    recs.append((q, int(i), int(d["iter"].ravel()[i]), d["F"].ravel()[i], d["C"].ravel()[i],
                                 d["S"].ravel()[i], d["snr"].ravel()[i]))
                per_plane.append(d if keep_planes else None)
        rec = np.array(recs, dtype=[("plane", "i2"), ("pix", "i4"), ("iter", "i2"), ("f", "f8"), ("c", "f8"),
                                    ("s", "f8"), ("snr", "f8")]) if recs else \
            np.zeros(0, dtype=[("plane", "i2"), ("pix", "i4"), ("iter", "i2"), ("f", "f8"), ("c", "f8"),
                               ("s", "f8"), ("snr", "f8")])
        upos, upl, us = dedupe(rec["pix"], rec["plane"], rec["snr"], p["Dy"], p["Dx"], p["r_dedupe"])
        out = dict(rec=rec, upos=upos, uplane=upl, usnr=us)
        if keep_planes:
            out["planes"] = per_plane
        return out

    def backfill(self, cube, ok, t: int):
        """O11, backward fill ("we backward fill the catalog ... add a pre-specified number of
        timesteps to the catalog and measure from cached images"): every slot born at t gets, for each cached
        frame tau in [t - n_back, t - 1] whose ring column still belongs to tau, the O9 flux of that frame at
        the slot's pixel.  Then frame t joins the cache."""
        if self.n_back <= 0:
            return
        tb = self.table
        new = np.flatnonzero((tb.active != 0) & (tb.born == t))
        if new.size:
            pix = tb.cpix[new]
            for (tau, c_tau, ok_tau) in self.history:
                if tau < t - self.n_back or tau >= t or tb.meta_t[tau % tb.T] != tau:
                    continue
                f = measure_flux(c_tau, ok_tau, self.W, pix, self.p["r_flux"])
                tb.ring[new, tau % tb.T, :] = f
        self.history.append((t, np.array(cube, dtype=np.float32, copy=True), np.array(ok, dtype=np.uint8, copy=True)))
        if len(self.history) > self.n_back:
            self.history.pop(0)

    def front(self, cube, keep_planes: bool = False):
        """The part of a step that has no memory (QC, per-plane detection, duplicate filter): (stats, band_ok, det).
        Frames are independent here, so a test harness may evaluate several frames at once and
        hand each result to step(pre=...).  Not with eq. A.2 on: that state is a recurrence over the frames."""
        assert self.rq is None, "the running per-pixel QC carries state from frame to frame"
        stats, ok = self.cube_qc(cube)
        return stats, ok, self.detect(cube, ok, keep_planes)

    def step(self, cube, t: int, keep_planes: bool = False, pre=None) -> dict:
        """One frame through the whole path.  pre: the result of front(cube), if it was evaluated beforehand."""
        p = self.p
        if pre is not None:
            stats, ok, det = pre
        else:
            stats, ok = self.cube_qc(cube)
            det = self.detect(cube, ok, keep_planes)
        cand, act_s, act_p = self.table.associate(det["upos"], t, int(ok[p["B"]]))
        flux = measure_flux(cube, ok, self.W, act_p, p["r_flux"])
        self.table.append(act_s, flux, ok, t)
        self.backfill(cube, ok, t)
        det.update(zeta_cnt=self.zeta_cnt.copy(), zeta_near=(self.rq.near.copy() if self.rq is not None else None))
        det.update(stats=stats, band_ok=ok, cand_idx=cand, act_slots=act_s, act_pix=act_p, flux=flux)
        return det


# ---------------------------------------------------------------------------------------------------
# O13 / O14: what the parameter-inference network is fed with ("x is a dynamic spectrum that we
# obtained from the image processing steps"; :197-210 eqs. 19-21, the simulated dispersed pulses it is trained on).
C_DM = 4148.806  # s MHz^2 cm^3 / pc (eq. 20, :206; R19)


def export_dynspec(table: "CandidateTable", slots, t_last: int, sigma=None) -> np.ndarray:
    """O13 -> [n][B][T_ring] float32: the time-ordered dynamic spectra (O10 view) of the given slots, each band
    divided by its noise sigma ("A ... in standard deviations of the noise", :208), samples that do not exist
    (NaN: before birth, rejected columns outside the ring) set to 0."""
    out = np.zeros((len(slots), table.B, table.T), dtype=np.float32)
    sg = np.ones(table.B, np.float64) if sigma is None else np.asarray(sigma, np.float64)
    sg = np.where(sg > 0, sg, 1.0)
    for i, s in enumerate(slots):
        ds = table.dynspec(int(s), t_last).astype(np.float64)
        ds = ds / sg[:, None]
        out[i] = np.where(np.isnan(ds), 0.0, ds).astype(np.float32)
    return out


def simulate_pulses(theta, nu, nu0: float, T: int, dt: float = 1.0) -> np.ndarray:
    """O14, eqs. 19-21 -> [n][B][T] float64.  theta rows: (t0 [steps], w [steps], DM [pc/cm^3], A, alpha).
    t_nu = t0 + C_DM DM (nu^-2 - nu0^-2) / dt  (eq. 20, nu in MHz, dt seconds per step);
    f = exp[-1/2 ((t - t_nu)/w)^2]  (eq. 19 with the 1/2 that its own "w = 16 <-> FWHM 37.67" implies, R18);
    I = A (nu/nu0)^alpha f  (eq. 21)."""
    theta = np.asarray(theta, np.float64).reshape(-1, 5)
    nu = np.asarray(nu, np.float64)
    t = np.arange(T, dtype=np.float64)
    out = np.zeros((theta.shape[0], nu.size, T))
    for i, (t0, w, dm, A, al) in enumerate(theta):
        for b, v in enumerate(nu):
            tn = t0 + C_DM * dm * (v ** -2 - nu0 ** -2) / dt
            out[i, b] = A * (v / nu0) ** al * np.exp(-0.5 * ((t - tn) / w) ** 2)
    return out
