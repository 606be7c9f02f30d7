"""-m gpu: parity at the extents of SURVEY.md 8(d)'s config table (the short cases are in test_gpu_parity.py; this file
sorts after it so that `-x -q` meets them first).

  config 2: all 300 frames;
  config 3: 64 frames that include every RFI frame of the first 200, one lane and eight lanes in flight;
  config 4: every 4th of the first 32 frames, four lanes in flight;
  config 5: a 160-frame flux / ring prefix (> T_ring = 128: wrap-around) with all 10 000 forced positions, and
            detection every 8th frame.

The oracle's memoryless front (QC + detection + duplicate filter) is evaluated for several frames at once on the host's
cores (oracle.OraclePipeline.front; the C++ oracle is called through ctypes, which releases the interpreter lock);
association, flux and rings then run in frame order.  Oracle runs use the rows-then-columns form of the window sums
(direct = False, reading R26, pinned against the direct form in test_oracle_pins.py); the direct form meets the kernel
in test_gpu_parity.py (config 1, one config-2 frame, the ragged case)."""
import os
from concurrent.futures import ThreadPoolExecutor

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle as O
from paper_2103_15418_b200 import synth
import parity

WORKERS = max(2, min(12, (os.cpu_count() or 4) - 1))


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available()
    return torch


def _make(cfg, n_lanes=1, **kw):
    from paper_2103_15418_b200.binding import LPF
    s = synth.CubeStream(cfg)
    p = synth.default_params(cfg)
    p.update(kw)
    p["n_lanes"] = n_lanes
    lpf = LPF(p, s.mask)
    assert lpf.plan()["fused"]
    return s, p, lpf


def _fronts(s, pipe, ts):
    """{t: (cube, front(cube))} for the frames ts, evaluated WORKERS at a time."""
    def one(t):
        cube = s.frame(t)
        return t, cube, pipe.front(cube)
    with ThreadPoolExecutor(WORKERS) as ex:
        return {t: (cube, pre) for t, cube, pre in ex.map(one, ts)}


def _chunks(seq, n):
    seq = list(seq)
    return [seq[i:i + n] for i in range(0, len(seq), n)]


def _run_in_flight(torch, lpf, s, p, pipe, ts, lanes, tag):
    """Frames ts through lpf_process_frame, `lanes` of them in flight on separate streams; every lane's result against
    the oracle.  Returns the number of logged ties."""
    streams = [torch.cuda.Stream() for _ in range(lanes)]
    ties = 0
    for chunk in _chunks(ts, 4 * lanes):
        pre = _fronts(s, pipe, chunk)
        for group in _chunks(chunk, lanes):
            dc = [torch.from_numpy(pre[t][0]).cuda() for t in group]
            torch.cuda.synchronize()
            for i, t in enumerate(group):
                lpf.process_frame(dc[i], t, lane=i, stream=streams[i])
            torch.cuda.synchronize()
            for i, t in enumerate(group):
                cube, fr = pre[t]
                o = pipe.step(cube, t, pre=fr)
                r = parity.check_frame(lpf.frame_view(i), o, pipe, cube, f"{tag} t={t}")
                assert r["in_sync"], f"{tag} t={t}: chain lost sync after a tie: {parity.TIES[-3:]}"
                ties += r["n_ties"]
    return ties


def _dynspecs_equal(lpf, pipe, slots, t_last):
    for slot in slots:
        a = lpf.get_dynspec(int(slot), t_last).cpu().numpy(); b = pipe.table.dynspec(int(slot), t_last)
        assert np.array_equal(np.isnan(a), np.isnan(b)) and np.array_equal(a[~np.isnan(a)], b[~np.isnan(b)]), slot


def test_config2_all_frames(torch_cuda):
    s, p, lpf = _make(2)
    pipe = O.OraclePipeline(p, s.mask, direct=False)
    ties = _run_in_flight(torch_cuda, lpf, s, p, pipe, range(300), 1, "cfg2 all")
    assert ties <= 2          # none expected on config 2
    act = np.flatnonzero(pipe.table.active)
    assert act.size > 100
    _dynspecs_equal(lpf, pipe, act[:: max(1, act.size // 40)], 299)
    assert lpf.counters()["dropped_records"] == 0 and lpf.counters()["dropped_detections"] == 0
    lpf.close()


def _config3_frames():
    s = synth.CubeStream(3)
    rfi = [t for t in range(200) if s.rfi(t)]
    want = set(rfi) | {t + 1 for t in rfi} | {0, 1, 2, 3}
    t = 4
    while len(want) < 64:
        want.add(t); t += 3
    return sorted(want), rfi


@pytest.mark.parametrize("lanes", [1, 8])
def test_config3_64_frames_with_every_rfi_frame(torch_cuda, lanes):
    ts, rfi = _config3_frames()
    assert len(ts) >= 64 and len(rfi) >= 5
    s, p, lpf = _make(3, n_lanes=lanes)
    pipe = O.OraclePipeline(p, s.mask, direct=False)
    ties = _run_in_flight(torch_cuda, lpf, s, p, pipe, ts, lanes, f"cfg3 x{lanes}")
    assert ties <= 10         # O(10) over ALL of config 3
    # QC flagged exactly the injected bands of every RFI frame (check_frame has compared band_ok with the oracle)
    for t in rfi:
        cube = s.frame(t)
        _, ok = pipe.cube_qc(cube)
        assert [b for b in range(p["B"]) if not ok[b]] == s.truth_rfi_bands(t), t
    act = np.flatnonzero(pipe.table.active)
    _dynspecs_equal(lpf, pipe, act[:: max(1, act.size // 30)], ts[-1])
    lpf.close()


def test_config4_every_4th_frame_four_lanes(torch_cuda):
    s, p, lpf = _make(4, n_lanes=4)
    pipe = O.OraclePipeline(p, s.mask, direct=False)
    ties = _run_in_flight(torch_cuda, lpf, s, p, pipe, range(0, 32, 4), 4, "cfg4 x4")
    assert ties <= 4
    lpf.close()


def test_config5_flux_ring_prefix_and_detection(torch_cuda):
    """All 10 000 forced positions x 64 bands over 160 frames (T_ring = 128: the ring wraps): fluxes and ring contents
    bit-exact through lpf_measure_flux / lpf_append_dynspec; every 8th frame also goes through the whole path on a
    second context."""
    torch = torch_cuda
    from paper_2103_15418_b200.binding import LPF
    s = synth.CubeStream(5)
    p = synth.default_params(5)
    assert p["T_ring"] == 128 and s.forced_pix.size == 10000
    lpf = LPF(p, s.mask)
    slots = lpf.add_candidates(s.forced_pix).cpu().numpy()
    tb = O.CandidateTable(p["n_cand_max"], p["T_ring"], p["B"], p["Dx"], p["r_assoc"], p["n_forget"])
    assert np.array_equal(tb.add_forced(s.forced_pix), slots)
    fp = s.forced_pix.astype(np.int32)
    pos_d = torch.from_numpy(fp).cuda(); slots_d = torch.from_numpy(slots.astype(np.int32)).cuda()
    n_d = torch.tensor([fp.size], dtype=torch.int32, device="cuda")
    det_lpf = LPF(p, s.mask)
    det_lpf.add_candidates(s.forced_pix)
    det_pipe = O.OraclePipeline(p, s.mask, direct=False)
    det_pipe.table.add_forced(s.forced_pix)
    ok = np.ones(p["B"] + 1, np.uint8)

    def one(t):
        cube = s.frame(t)
        okt = ok.copy()
        if t % 37 == 5:
            okt[t % p["B"]] = 0            # a rejected band now and then: its flux is 0
        return t, cube, okt, O.measure_flux(cube, okt, s.mask, fp, p["r_flux"]), (det_pipe.front(cube) if t % 8 == 0 else None)

    ties = 0
    for chunk in _chunks(range(160), WORKERS):
        with ThreadPoolExecutor(WORKERS) as ex:
            res = list(ex.map(one, chunk))
        for t, cube, okt, flux_o, fr in res:
            cube_d = torch.from_numpy(cube).cuda(); ok_d = torch.from_numpy(okt).cuda()
            flux_d = lpf.measure_flux(cube_d, ok_d, pos_d, n_d)
            lpf.append_dynspec(slots_d, n_d, flux_d, ok_d, t)
            tb.append(slots, flux_o, okt, t)
            assert np.array_equal(flux_d.cpu().numpy(), flux_o), t
            if fr is not None:
                o = det_pipe.step(cube, t, pre=fr)
                det_lpf.process_frame(cube_d, t)
                r = parity.check_frame(det_lpf.frame_view(0), o, det_pipe, cube, f"cfg5 t={t}")
                assert r["in_sync"]
                ties += r["n_ties"]
    assert ties <= 4
    rng = np.random.default_rng(1)
    for slot in rng.choice(fp.size, 64, replace=False):
        a = lpf.get_dynspec(int(slot), 159).cpu().numpy(); b = tb.dynspec(int(slot), 159)
        assert not np.isnan(a).any()              # 160 > T_ring: every column has been written
        assert np.array_equal(a, b), slot
    lpf.close(); det_lpf.close()
