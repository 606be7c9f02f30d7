"""Pins for the seeded input generator (paper_2103_15418_b200/synth.py).

The generator serves both the oracle and the CUDA path, so it is pinned to what
the paper / mathematics fix: the dispersion-delay closed form (PAPER.md:203-206,
eq. 20), the eq.-19 profile width consistency, the power-law
closed forms and the horizon-mask pixel counts (SURVEY.md 8(c) "generator").
"""
import os

import numpy as np
import pytest

from paper_2103_15418_b200 import synth

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def test_dispersion_delay_golden():
    for line in open(os.path.join(GOLD, "dispersion_delays.txt")):
        if line.startswith("#") or not line.strip():
            continue
        dm, nu, ref, want, tol = line.split()
        got = synth.dispersion_delay_s(float(dm), float(nu), float(ref))
        assert abs(got - float(want)) <= float(tol) + 1e-4 * abs(float(want)), line


def test_dispersion_constant_matches_north_star():
    # north_star quotes 4.149e3; PAPER.md:206 prints 4148.806 -> agree to 1e-4
    assert abs(synth.C_DM - 4.149e3) / 4.149e3 < 1e-4


def test_profile_fwhm_consistency():
    # "w ... 16, corresponding to a maximum FWHM of 37.67 time-steps"
    # -> profile is exp[-1/2 ((t-t0)/w)^2]  (reading R18)
    assert abs(2 * np.sqrt(2 * np.log(2)) * 16 - 37.67) < 1e-2      # paper truncates 37.677
    assert abs(2 * np.sqrt(np.log(2)) * 16 - 37.67) > 10             # eq. 19 as printed (no 1/2) does not fit
    s = synth.CubeStream(2)
    i = 0
    w = s.transients["w"][i]
    t0 = s.transients["t0"][i] + s.delay[i, 0]
    # half maximum at t0 +- w sqrt(2 ln 2)
    th = t0 + w * np.sqrt(2 * np.log(2))
    arg = (th - s.transients["t0"][i] - s.delay[i, 0]) / w
    assert abs(np.exp(-0.5 * arg ** 2) - 0.5) < 1e-12


def test_power_law_closed_forms():
    rng = np.random.default_rng(1)
    S = synth.power_law_snr(rng, 400000, 3.0, 50.0)
    a = -0.5
    med = (3 ** a + 0.5 * (50 ** a - 3 ** a)) ** (1 / a)
    frac10 = (10 ** a - 50 ** a) / (3 ** a - 50 ** a)
    assert abs(med - 7.7424) < 1e-3 and abs(frac10 - 0.4010) < 1e-3
    assert abs(np.median(S) - med) < 0.05
    assert abs((S > 10).mean() - frac10) < 0.005
    assert S.min() >= 3.0 and S.max() <= 50.0


@pytest.mark.parametrize("n,count", [(1024, 667064), (2048, 2668400)])
def test_horizon_mask_counts(n, count):
    assert int(synth.horizon_mask(n).sum()) == count


def test_source_sigma():
    assert abs(synth.SIGMA_SRC - 0.849322) < 1e-6


def test_config1_content():
    s = synth.CubeStream(1)
    assert s.mask is None
    assert s.c.B == 4 and s.c.D == 64 and s.c.T == 32
    # noiseless template: 10 sigma peak at (row, col) = (20, 37)  (reading R24)
    assert np.unravel_index(np.argmax(s.template), s.template.shape) == (20, 37)
    assert abs(s.template[20, 37] - 10.0) < 1e-6
    f0, f0b = s.frame(0), s.frame(0)
    assert f0.dtype == np.float32 and f0.shape == (4, 64, 64) and f0.flags.c_contiguous
    assert np.array_equal(f0, f0b)              # seeded
    assert not np.array_equal(f0, s.frame(1))   # frame noise differs
    assert abs(float((f0 - s.template).std()) - 1.0) < 0.02


def test_config2_bands_and_transients():
    s = synth.CubeStream(2)
    f = s.c.freqs_mhz
    assert f.size == 16 and abs(f[0] - 57.0) < 1e-12 and abs(f[7] - 58.3671875) < 1e-9
    assert abs(f[8] - 61.7) < 1e-12 and abs(f[15] - 63.0671875) < 1e-9
    assert s.steady["y"].size == 200 and s.transients["y"].size == 10
    assert (s.transients["dm"] >= 0).all() and (s.transients["dm"] <= 30).all()
    # lower frequencies arrive later and the delay is the closed form
    assert (np.diff(s.delay, axis=1)[:, :7] < 0).all()
    i = int(np.argmax(s.transients["dm"]))
    want = synth.C_DM * s.transients["dm"][i] * (57.0 ** -2 - 63.1 ** -2)
    assert abs(s.delay[i, 0] - want) < 1e-9
    # the per-band peak time of the injected profile is t0 + dt_b (integer sampling: +-1 step)
    tt = np.arange(s.c.T)
    amps = np.stack([s.transient_amplitudes(int(t))[i] for t in tt])  # [T, B]
    tpk = tt[np.argmax(amps, axis=0)]
    assert np.all(np.abs(tpk - (s.transients["t0"][i] + s.delay[i])) <= 1.0)


def test_config3_mask_noise_rfi():
    s = synth.CubeStream(3)
    assert s.mask is not None and int(s.mask.sum()) == 667064
    c = (1024 - 1) / 2
    assert abs(s.sigma_map[int(c), int(c)] - 1.0) < 0.01
    edge = s.sigma_map[512, 512 + 460]
    assert abs(edge - 3.0) < 0.02
    # RFI frames: about 5 % of frames, 1..4 bands each
    n_rfi = sum(1 for t in range(600) if s.rfi(t))
    assert 10 <= n_rfi <= 55
    t_bad = next(t for t in range(600) if s.rfi(t))
    assert 1 <= len(s.truth_rfi_bands(t_bad)) <= 4


def test_config5_forced_positions():
    s = synth.CubeStream(5)
    assert s.c.B == 64 and abs(s.c.freqs_mhz[0] - 50) < 1e-12 and abs(s.c.freqs_mhz[-1] - 80) < 1e-12
    assert s.forced_pix.size == 10000
    assert s.mask.ravel()[s.forced_pix].all()
    d = synth.dispersion_delay_s(100.0, s.c.freqs_mhz, 80.0)
    assert abs(d[0] - 101.1271) < 1e-3 and abs(d[31] - 34.0949) < 1e-3 and d[63] == 0.0
