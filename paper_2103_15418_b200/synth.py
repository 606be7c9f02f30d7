"""Seeded synthetic image-cube streams shaped like the paper's AARTFAAC workloads.

This module is the ONE piece shared by the CPU oracle (``oracle/``) and the CUDA
path: it only *makes inputs*.  It holds none of the method's arithmetic (no
statistics, no convolution, no thresholding, no flux extraction) and imports
neither side.  NumPy only.

What it stands in for: the paper measures on AARTFAAC all-sky cubes of
16 x 1024 x 1024 and on simulated skies.
Neither the survey data nor the paper's foreground map / PSF recipe is available,
so the five workloads below follow BASELINE.json's ``configs``.

Recipe (all configs):
  * static content is drawn from ``default_rng([seed, cfg, 0])``,
    frame ``t`` noise from ``default_rng([seed, cfg, 1, t])``, RFI decisions
    from ``default_rng([seed, cfg, 2, t])``;
  * a point source is a circular Gaussian of FWHM 2 px (sigma = 0.849322 px)
    centred on an integer pixel, stamped out to radius 5 px, amplitude =
    SNR x the local noise sigma, identical in every band (flat spectrum);
  * a dispersed transient has the time profile A exp[-1/2 ((t - t0 - dt_b)/w)^2]
    sampled at integer seconds (eq. 19 with the 1/2 that the text's
    "w=16 <-> FWHM 37.67" implies, reading R18) with the per-band delay
    dt_b = C_DM DM (nu_b^-2 - nu_ref^-2), C_DM = 4148.806 s MHz^2 cm^3/pc
    (eq. 20, reading R19);
  * horizon mask: valid iff (y-c)^2 + (x-c)^2 <= (0.45 N)^2, c = (N-1)/2; masked
    pixels are exactly 0; noise sigma(r) = 1 + 2 min(r / 0.45N, 1) where stated.
"""
from __future__ import annotations

import dataclasses
from typing import Dict, List, Optional

import numpy as np

C_DM = 4148.806  # s MHz^2 cm^3 / pc
FWHM_PX = 2.0
SIGMA_SRC = FWHM_PX / (2.0 * np.sqrt(2.0 * np.log(2.0)))  # 0.849322
STAMP_R = 5


def dispersion_delay_s(dm: float, nu_mhz, nu_ref_mhz: float):
    """Cold-plasma dispersion delay in seconds, eq. 20."""
    nu = np.asarray(nu_mhz, dtype=np.float64)
    return C_DM * dm * (nu ** -2.0 - float(nu_ref_mhz) ** -2.0)


def aartfaac_bands_mhz() -> np.ndarray:
    """Two groups of 8 contiguous 195.3125 kHz subbands (BASELINE.json config 2)."""
    i = np.arange(8, dtype=np.float64)
    return np.concatenate([57.0 + 0.1953125 * i, 61.7 + 0.1953125 * i])


def power_law_snr(rng, n: int, lo: float, hi: float, index: float = -1.5) -> np.ndarray:
    """Draw from dN/dS ~ S^index on [lo, hi] by inverting the CDF."""
    a = index + 1.0
    u = rng.random(n)
    return (lo ** a + u * (hi ** a - lo ** a)) ** (1.0 / a)


def horizon_mask(n: int) -> np.ndarray:
    c = (n - 1) / 2.0
    yy, xx = np.mgrid[:n, :n]
    return (((yy - c) ** 2 + (xx - c) ** 2) <= (0.45 * n) ** 2).astype(np.uint8)


def noise_sigma_map(n: int) -> np.ndarray:
    c = (n - 1) / 2.0
    yy, xx = np.mgrid[:n, :n]
    r = np.sqrt((yy - c) ** 2 + (xx - c) ** 2)
    return 1.0 + 2.0 * np.minimum(r / (0.45 * n), 1.0)


@dataclasses.dataclass
class StreamConfig:
    name: str
    cfg: int
    D: int
    B: int
    T: int
    freqs_mhz: np.ndarray
    nu_ref_mhz: float
    masked: bool = False
    radial_noise: bool = False
    n_steady: int = 0
    steady_snr: tuple = (3.0, 50.0)
    n_transient: int = 0
    dm_range: tuple = (0.0, 0.0)
    width_range: tuple = (1.0, 1.0)
    tr_snr: tuple = (5.0, 20.0)
    rfi_prob: float = 0.0
    n_forced: int = 0
    n_lanes: int = 1
    fixed_sources: Optional[list] = None  # [(y, x, snr)]


def _configs() -> Dict[int, StreamConfig]:
    b16 = aartfaac_bands_mhz()
    return {
        1: StreamConfig("tiny_64x64x4", 1, 64, 4, 32, b16[:4].copy(), 63.1,
                        fixed_sources=[(20, 37, 10.0)]),
        2: StreamConfig("small_256x256x16", 2, 256, 16, 300, b16, 63.1,
                        n_steady=200, n_transient=10, dm_range=(0.0, 30.0),
                        width_range=(1.0, 5.0), tr_snr=(5.0, 20.0)),
        3: StreamConfig("allsky_1024x1024x16", 3, 1024, 16, 600, b16, 63.1,
                        masked=True, radial_noise=True, n_steady=2000, n_transient=50,
                        dm_range=(0.0, 60.0), width_range=(1.0, 10.0), tr_snr=(5.0, 30.0),
                        rfi_prob=0.05),
        4: StreamConfig("stress_2048x2048x16", 4, 2048, 16, 256, b16, 63.1,
                        masked=True, radial_noise=True, n_steady=8000, n_transient=200,
                        dm_range=(0.0, 60.0), width_range=(1.0, 10.0), tr_snr=(5.0, 30.0),
                        n_lanes=4),
        5: StreamConfig("wideband_1024x1024x64", 5, 1024, 64, 512,
                        np.linspace(50.0, 80.0, 64), 80.0,
                        masked=True, radial_noise=True, n_steady=5000, n_transient=500,
                        dm_range=(0.0, 100.0), width_range=(1.0, 10.0), tr_snr=(5.0, 30.0),
                        n_forced=10000),
    }


CONFIGS = _configs()


def default_params(cfg: int, bg: str = "box", n_iter: int = 1) -> dict:
    """Parameter set of SURVEY.md section 8 (kappa=5, 5x5 max filter, sigma_mf=0.85 ...).

    Plain dict of numbers; both sides turn it into their own parameter struct.
    """
    c = CONFIGS[cfg]
    p = dict(
        B=c.B, Dy=c.D, Dx=c.D,
        kappa=5.0, k_max=2, eps_rel=1e-5,
        sigma_mf=0.85, k_mf=3,
        bg_kernel=1 if bg == "box" else 0,
        s_bg=8.0, k_bg=12 if bg == "box" else 16,
        n_iter=n_iter, detect_sum_plane=1,
        qc_tau=5.0, qc_clip=3.0,
        r_flux=1, r_dedupe=2, r_assoc=3, n_forget=10,
        T_ring=128,
        n_cand_max={1: 64, 2: 2048, 3: 8192, 4: 32768, 5: 32768}[cfg],
        max_det={1: 1024, 2: 16384, 3: 131072, 4: 524288, 5: 524288}[cfg],
        n_lanes=c.n_lanes,
        n_back=0,
        zeta_thr=0.0, zeta_nmax=0, zeta_window=64, zeta_warm=16,
    )
    return p


class CubeStream:
    """A seeded stream of image cubes X_t in R^{B x D x D}."""

    def __init__(self, cfg: int, seed: int = 0):
        self.c = CONFIGS[cfg]
        self.cfg = cfg
        self.seed = seed
        c = self.c
        D = c.D
        rng = np.random.default_rng([seed, cfg, 0])
        self.mask = horizon_mask(D) if c.masked else None
        self.sigma_map = (noise_sigma_map(D) if c.radial_noise else np.ones((D, D))).astype(np.float32)
        if self.mask is not None:
            self.sigma_map = self.sigma_map * self.mask
        valid_idx = np.flatnonzero(self.mask.ravel()) if self.mask is not None else None

        def draw_pix(n):
            if valid_idx is None:
                p = rng.integers(0, D * D, size=n)
            else:
                p = valid_idx[rng.integers(0, valid_idx.size, size=n)]
            return p // D, p % D

        # steady sources
        if c.fixed_sources:
            ys = np.array([s[0] for s in c.fixed_sources])
            xs = np.array([s[1] for s in c.fixed_sources])
            snr = np.array([s[2] for s in c.fixed_sources], dtype=np.float64)
        else:
            ys, xs = draw_pix(c.n_steady)
            snr = power_law_snr(rng, c.n_steady, *c.steady_snr)
        self.steady = dict(y=ys.astype(np.int64), x=xs.astype(np.int64), snr=snr)
        amp = snr * self.sigma_map[ys, xs].astype(np.float64) if ys.size else snr
        self.steady["amp"] = amp
        tmpl = np.zeros((D, D), dtype=np.float64)
        for y, x, a in zip(ys, xs, amp):
            self._stamp(tmpl, int(y), int(x), float(a))
        if self.mask is not None:
            tmpl *= self.mask
        self.template = tmpl.astype(np.float32)

        # dispersed transients
        nt = c.n_transient
        ty, tx = draw_pix(nt) if nt else (np.zeros(0, int), np.zeros(0, int))
        self.transients = dict(
            y=ty.astype(np.int64), x=tx.astype(np.int64),
            dm=rng.uniform(*c.dm_range, size=nt),
            w=rng.uniform(*c.width_range, size=nt),
            snr=rng.uniform(*c.tr_snr, size=nt),
            t0=rng.uniform(0.1 * c.T, 0.9 * c.T, size=nt),
        )
        self.transients["amp"] = (self.transients["snr"] *
                                  (self.sigma_map[ty, tx].astype(np.float64) if nt else 1.0))
        # per-band delay table [nt, B]
        self.delay = np.stack([dispersion_delay_s(dm, c.freqs_mhz, c.nu_ref_mhz)
                               for dm in self.transients["dm"]]) if nt else np.zeros((0, c.B))

        # forced candidate positions (config 5): true positions + uniform valid pixels
        if c.n_forced:
            true_pix = np.concatenate([ys * D + xs, ty * D + tx])
            n_extra = c.n_forced - true_pix.size
            ey, ex = draw_pix(n_extra)
            self.forced_pix = np.concatenate([true_pix, ey * D + ex]).astype(np.int32)
        else:
            self.forced_pix = np.zeros(0, dtype=np.int32)

        # the stamp (unit amplitude), reused for transients
        r = STAMP_R
        yy, xx = np.mgrid[-r:r + 1, -r:r + 1]
        self._unit_stamp = np.exp(-(yy ** 2 + xx ** 2) / (2.0 * SIGMA_SRC ** 2))

    # ------------------------------------------------------------------
    @staticmethod
    def _stamp(img, y, x, a):
        D0, D1 = img.shape
        r = STAMP_R
        y0, y1 = max(0, y - r), min(D0, y + r + 1)
        x0, x1 = max(0, x - r), min(D1, x + r + 1)
        yy, xx = np.mgrid[y0:y1, x0:x1]
        img[y0:y1, x0:x1] += a * np.exp(-((yy - y) ** 2 + (xx - x) ** 2) / (2.0 * SIGMA_SRC ** 2))

    def transient_amplitudes(self, t: int) -> np.ndarray:
        """[n_transient, B] amplitudes at integer time t."""
        tr = self.transients
        if tr["y"].size == 0:
            return np.zeros((0, self.c.B))
        arg = (t - tr["t0"][:, None] - self.delay) / tr["w"][:, None]
        return tr["amp"][:, None] * np.exp(-0.5 * arg ** 2)

    def rfi(self, t: int):
        """RFI decisions for frame t: list of (band, kind, rows) ; kind 0 = noise x10, 1 = stripes."""
        c = self.c
        if c.rfi_prob <= 0.0:
            return []
        rng = np.random.default_rng([self.seed, self.cfg, 2, t])
        if rng.random() >= c.rfi_prob:
            return []
        nb = int(rng.integers(1, 5))
        bands = rng.choice(c.B, size=nb, replace=False)
        out = []
        for b in bands:
            kind = int(rng.integers(0, 2))
            if kind == 0:
                out.append((int(b), 0, None))
            else:
                nrow = int(rng.integers(1, 9))
                # rows through the valid disc
                lo, hi = int(0.1 * c.D), int(0.9 * c.D)
                rows = rng.integers(lo, hi, size=nrow)
                out.append((int(b), 1, np.unique(rows)))
        return out

    def frame(self, t: int) -> np.ndarray:
        """Cube at time step t: float32 [B, D, D], C-contiguous."""
        c = self.c
        D, B = c.D, c.B
        rng = np.random.default_rng([self.seed, self.cfg, 1, t])
        cube = rng.standard_normal((B, D, D), dtype=np.float32)
        rfi = self.rfi(t)
        scale = np.ones(B, dtype=np.float32)
        for (b, kind, rows) in rfi:
            if kind == 0:
                scale[b] = 10.0
        cube *= (self.sigma_map[None, :, :] * scale[:, None, None])
        cube += self.template[None, :, :]
        amps = self.transient_amplitudes(t)
        tr = self.transients
        r = STAMP_R
        for i in range(amps.shape[0]):
            a = amps[i]
            if a.max() < 1e-4 * max(tr["amp"][i], 1e-30):
                continue
            y, x = int(tr["y"][i]), int(tr["x"][i])
            y0, y1 = max(0, y - r), min(D, y + r + 1)
            x0, x1 = max(0, x - r), min(D, x + r + 1)
            st = self._unit_stamp[y0 - y + r:y1 - y + r, x0 - x + r:x1 - x + r]
            add = a[:, None, None] * st[None]
            if self.mask is not None:
                add = add * self.mask[None, y0:y1, x0:x1]
            cube[:, y0:y1, x0:x1] += add.astype(np.float32)
        for (b, kind, rows) in rfi:
            if kind == 1:
                cube[b, rows, :] += 20.0 * self.sigma_map[rows, :]
        return np.ascontiguousarray(cube)

    def truth_rfi_bands(self, t: int) -> List[int]:
        return sorted({b for (b, _, _) in self.rfi(t)})
