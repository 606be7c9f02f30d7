"""-m gpu: the CUDA path (through the C-ABI) against the CPU oracle, element by element,
on the five BASELINE.json configs (SURVEY.md 8(d) parity scope, sized to finish in minutes)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle as O
from paper_2103_15418_b200 import synth
import parity


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available()
    return torch


def _make(cfg, torch, **kw):
    """Context for a config.  general=True forces the multi-kernel general path (lpf_params.force_general);
    otherwise box/K=12/n_iter=1 contexts take the fused single-pass kernel."""
    from paper_2103_15418_b200.binding import LPF
    s = synth.CubeStream(cfg)
    bg = kw.pop("bg", "box"); n_iter = kw.pop("n_iter", 1); general = kw.pop("general", False)
    p = synth.default_params(cfg, bg=bg, n_iter=n_iter)
    p.update(kw)
    p["force_general"] = 1 if general else 0
    lpf = LPF(p, s.mask)
    want_fused = (not general) and bg == "box" and n_iter == 1 and p["k_bg"] == 12 and p["k_mf"] == 3
    assert lpf.plan()["fused"] == want_fused, lpf.plan()
    return s, p, lpf


def _run_chain(torch, s, p, lpf, frames, direct=False, via="calls", tag=""):
    pipe = O.OraclePipeline(p, s.mask, direct=direct)
    worst_z = 0.0; ties = 0
    for t in frames:
        cube = s.frame(t)
        cube_d = torch.from_numpy(cube).cuda()
        o = pipe.step(cube, t)
        if via == "calls":
            g = parity.gpu_step_by_calls(lpf, cube_d, t)
        else:
            lpf.process_frame(cube_d, t)
            g = lpf.frame_view(0)
        r = parity.check_frame(g, o, pipe, cube, f"{tag} t={t}")
        assert r["in_sync"], f"{tag} t={t}: chain lost sync after a tie: {parity.TIES[-3:]}"
        worst_z = max(worst_z, r["zerr"]); ties += r["n_ties"]
    return pipe, worst_z, ties


# ------------------------------------------------------------------ config 1
@pytest.mark.parametrize("bg,n_iter,general", [("box", 1, False), ("box", 1, True), ("gauss", 1, True), ("box", 3, True),
                                               ("gauss", 3, True)])
def test_config1_all_frames(torch_cuda, bg, n_iter, general):
    s, p, lpf = _make(1, torch_cuda, bg=bg, n_iter=n_iter, general=general)
    pipe, wz, ties = _run_chain(torch_cuda, s, p, lpf, range(32), direct=True, via="calls", tag=f"cfg1 {bg} it{n_iter}")
    assert ties == 0
    # dynamic spectrum of the source's candidate: bit-exact, time ordered
    ds_g = lpf.get_dynspec(0, 31).cpu().numpy()
    ds_o = pipe.table.dynspec(0, 31)
    assert np.array_equal(np.isnan(ds_g), np.isnan(ds_o))
    assert np.array_equal(ds_g[~np.isnan(ds_g)], ds_o[~np.isnan(ds_o)])
    assert lpf.counters()["dropped_records"] == 0
    lpf.close()


def test_config1_process_frame_entry(torch_cuda):
    s, p, lpf = _make(1, torch_cuda)
    _run_chain(torch_cuda, s, p, lpf, range(8), via="frame", tag="cfg1 process_frame")
    lpf.close()


# ------------------------------------------------------------------ config 2
def test_config2_chain_box(torch_cuda):
    s, p, lpf = _make(2, torch_cuda)
    pipe, wz, ties = _run_chain(torch_cuda, s, p, lpf, range(40), via="frame", tag="cfg2 box")
    assert ties == 0
    # every active candidate's dynamic spectrum is bit-exact
    act = np.flatnonzero(pipe.table.active)
    assert act.size > 50
    for slot in act[:: max(1, act.size // 25)]:
        ds_g = lpf.get_dynspec(int(slot), 39).cpu().numpy(); ds_o = pipe.table.dynspec(int(slot), 39)
        assert np.array_equal(np.isnan(ds_g), np.isnan(ds_o)) and np.array_equal(ds_g[~np.isnan(ds_g)], ds_o[~np.isnan(ds_o)])
    lpf.close()


@pytest.mark.parametrize("bg,n_iter", [("box", 1), ("gauss", 1), ("box", 3), ("gauss", 3)])
def test_config2_variants(torch_cuda, bg, n_iter):
    s, p, lpf = _make(2, torch_cuda, bg=bg, n_iter=n_iter, general=True)
    _run_chain(torch_cuda, s, p, lpf, range(4), via="calls", tag=f"cfg2 {bg} it{n_iter}")
    lpf.close()


def test_config2_direct_definition_one_frame(torch_cuda):
    # the oracle's direct 2-D window form (no factorisation) on a full config-2 frame
    s, p, lpf = _make(2, torch_cuda)
    _run_chain(torch_cuda, s, p, lpf, [0], direct=True, tag="cfg2 direct")
    lpf.close()


# ------------------------------------------------------------------ config 3
def test_config3_frames_with_rfi(torch_cuda):
    s, p, lpf = _make(3, torch_cuda)
    t_bad = next(t for t in range(600) if s.rfi(t))
    frames = [0, t_bad, t_bad + 1] if t_bad > 0 else [0, 1]
    pipe = O.OraclePipeline(p, s.mask, direct=False)
    for t in frames:
        cube = s.frame(t)
        o = pipe.step(cube, t)
        lpf.process_frame(torch_cuda.from_numpy(cube).cuda(), t)
        g = lpf.frame_view(0)
        r = parity.check_frame(g, o, pipe, cube, f"cfg3 t={t}")
        assert r["in_sync"]
        if t == t_bad:   # QC must flag every injected band (and nothing else)
            bad = s.truth_rfi_bands(t)
            assert [b for b in range(p["B"]) if not o["band_ok"][b]] == bad
            assert [b for b in range(p["B"]) if not g["band_ok"][b]] == bad
    lpf.close()


@pytest.mark.parametrize("bg", ["gauss", "box"])
def test_config3_general_path_one_frame(torch_cuda, bg):
    s, p, lpf = _make(3, torch_cuda, bg=bg, general=True)
    _run_chain(torch_cuda, s, p, lpf, [0], via="frame", tag=f"cfg3 general {bg}")
    lpf.close()


# ------------------------------------------------------------------ config 4
def test_config4_four_lanes(torch_cuda):
    torch = torch_cuda
    s, p, lpf = _make(4, torch)
    assert p["n_lanes"] == 4
    cubes = [s.frame(t) for t in range(4)]
    dcubes = [torch.from_numpy(c).cuda() for c in cubes]
    streams = [torch.cuda.Stream() for _ in range(4)]
    torch.cuda.synchronize()
    for t in range(4):   # four frames in flight on separate CUDA streams
        lpf.process_frame(dcubes[t], t, lane=t, stream=streams[t])
    torch.cuda.synchronize()
    views = [lpf.frame_view(t) for t in range(4)]
    pipe = O.OraclePipeline(p, s.mask, direct=False)
    o0 = pipe.step(cubes[0], 0)
    r = parity.check_frame(views[0], o0, pipe, cubes[0], "cfg4 t=0")
    assert r["in_sync"]
    # frames 1..3: the association chain must have run in t order across lanes: same result as a
    # fresh single-lane context fed sequentially
    from paper_2103_15418_b200.binding import LPF
    p1 = dict(p); p1["n_lanes"] = 1
    seq = LPF(p1, s.mask)
    for t in range(4):
        seq.process_frame(dcubes[t], t)
        v = seq.frame_view(0)
        for k in ("band_ok", "upos", "cand_idx", "act_slots", "act_pix", "flux"):
            assert np.array_equal(v[k], views[t][k]), (t, k)
    seq.close(); lpf.close()


# ------------------------------------------------------------------ config 5
def test_config5_forced_flux_and_detection(torch_cuda):
    torch = torch_cuda
    s, p, lpf = _make(5, torch)
    slots = lpf.add_candidates(s.forced_pix).cpu().numpy()
    assert np.array_equal(slots, np.arange(10000))
    pipe = O.OraclePipeline(p, s.mask, direct=False)
    pipe.table.add_forced(s.forced_pix)
    cube = s.frame(0)
    o = pipe.step(cube, 0)
    lpf.process_frame(torch.from_numpy(cube).cuda(), 0)
    g = lpf.frame_view(0)
    r = parity.check_frame(g, o, pipe, cube, "cfg5 t=0")
    assert r["in_sync"] and g["flux"].shape[0] >= 10000 and g["flux"].shape[1] == 64
    lpf.close()


def test_config5_ring_wraparound(torch_cuda):
    # 64-channel rings with forced positions; T_ring shortened so that the wrap-around is reached in 20 frames
    torch = torch_cuda
    s = synth.CubeStream(5)
    p = synth.default_params(5); p["T_ring"] = 16
    from paper_2103_15418_b200.binding import LPF
    lpf = LPF(p, s.mask)
    n_forced = 2000
    fp = s.forced_pix[:n_forced]
    lpf.add_candidates(fp)
    tb = O.CandidateTable(p["n_cand_max"], 16, 64, p["Dx"], p["r_assoc"], p["n_forget"])
    slots = tb.add_forced(fp)
    pos_d = torch.from_numpy(fp.astype(np.int32)).cuda(); slots_d = torch.from_numpy(slots).cuda()
    n_d = torch.tensor([n_forced], dtype=torch.int32, device="cuda")
    rng = np.random.default_rng(0)
    for t in range(20):
        cube = s.frame(t)
        ok = np.ones(65, np.uint8)
        if t == 7:
            ok[5] = 0
        if t == 9:
            ok[64] = 0
        ok_d = torch.from_numpy(ok).cuda()
        cube_d = torch.from_numpy(cube).cuda()
        flux_d = lpf.measure_flux(cube_d, ok_d, pos_d, n_d)
        lpf.append_dynspec(slots_d, n_d, flux_d, ok_d, t)
        flux_o = O.measure_flux(cube, ok, s.mask, fp, p["r_flux"])
        tb.append(slots, flux_o, ok, t)
        assert np.array_equal(flux_d.cpu().numpy(), flux_o), t
    for slot in rng.choice(n_forced, 40, replace=False):
        a = lpf.get_dynspec(int(slot), 19).cpu().numpy(); b = tb.dynspec(int(slot), 19)
        assert np.array_equal(np.isnan(a), np.isnan(b)) and np.array_equal(a[~np.isnan(a)], b[~np.isnan(b)])
        assert not np.isnan(a).any()
    lpf.close()


# ------------------------------------------------------------------ edge cases
def test_edge_cases(torch_cuda):
    torch = torch_cuda
    from paper_2103_15418_b200.binding import LPF, LpfError
    # ragged sizes (not multiples of the tile, odd row length -> scalar load path), run-time radii
    rng = np.random.default_rng(21)
    Dy, Dx, B = 77, 93, 3
    p = synth.default_params(1); p.update(B=B, Dy=Dy, Dx=Dx, k_mf=2, k_bg=5, kappa=3.5, n_iter=2, n_cand_max=256, T_ring=4)
    W = (rng.random((Dy, Dx)) > 0.1).astype(np.uint8); W[:9, :11] = 0
    cube = rng.standard_normal((B, Dy, Dx)).astype(np.float32)
    cube[:, 40, 50] += 9.0; cube[:, 41, 50] += 6.0; cube[:, 5, 88] += 9.0
    cube *= W
    lpf = LPF(p, W)
    pipe = O.OraclePipeline(p, W, direct=True)
    for t in range(3):
        o = pipe.step(cube, t)
        g = parity.gpu_step_by_calls(lpf, torch.from_numpy(cube).cuda(), t)
        assert parity.check_frame(g, o, pipe, cube, f"ragged t={t}")["in_sync"]
    lpf.close()
    # constant cube: zero detections; all bands ok
    p = synth.default_params(1)
    lpf = LPF(p, None)
    for c in (0.0, 3.25, -1e6):
        cube = np.full((4, 64, 64), c, np.float32)
        g = parity.gpu_step_by_calls(lpf, torch.from_numpy(cube).cuda(), 0)
        assert g["ndets"] == 0 and g["upos"].size == 0 and g["band_ok"].all()
    # non-finite band is rejected, the rest of the frame is processed
    s = synth.CubeStream(1)
    cube = s.frame(0); cube[2, 10, 10] = np.nan
    pipe = O.OraclePipeline(p, None, direct=False)
    o = pipe.step(cube, 0)
    g = parity.gpu_step_by_calls(lpf, torch.from_numpy(cube).cuda(), 1)
    assert g["band_ok"].tolist() == [1, 1, 0, 1, 1] == o["band_ok"].tolist()
    assert np.array_equal(g["upos"], o["upos"]) and np.array_equal(g["flux"][:, 2], np.zeros(g["flux"].shape[0], np.float32))
    # rejected frame (majority of bands bad): no detections, zero fluxes, table unchanged
    cube = s.frame(1); cube[0, 3, 3] = np.inf; cube[1, 9, 9] = np.nan; cube[3, 1, 1] = -np.inf
    o = pipe.step(cube, 2)
    g = parity.gpu_step_by_calls(lpf, torch.from_numpy(cube).cuda(), 2)
    assert o["band_ok"][4] == 0 and g["band_ok"].tolist() == o["band_ok"].tolist()
    assert g["upos"].size == 0 and np.all(g["flux"] == 0) and np.array_equal(g["act_slots"], o["act_slots"])
    lpf.close()
    # capacity overflow is counted, not UB
    p2 = synth.default_params(1); p2["max_det"] = 2; p2["kappa"] = 1.0
    lpf = LPF(p2, None)
    g = parity.gpu_step_by_calls(lpf, torch.from_numpy(s.frame(0)).cuda(), 0)
    cnt = lpf.counters()
    assert g["ndets"] > 2 and len(g["rec"]) == 2 and cnt["dropped_records"] == g["ndets"] - 2 and cnt["truncated"]   # LPF_W_CAPACITY
    lpf.close()
    # argument errors
    bad = synth.default_params(1); bad["k_bg"] = 40
    with pytest.raises(LpfError):
        LPF(bad, None)
    # a forced position outside the image refuses the whole call on the device; the table stays as it was
    lpf = LPF(synth.default_params(1), None)
    n_pix = 64 * 64
    for wrong in (np.array([5, n_pix], np.int32), np.array([-1, 7], np.int32)):
        with pytest.raises(LpfError):
            lpf.add_candidates(wrong)
    slots = lpf.add_candidates(np.array([5, 7], np.int32)).cpu().numpy()
    assert slots.tolist() == [0, 1] and lpf.counters()["n_active"] == 2
    lpf.close()


def test_host_entry_point(torch_cuda):
    torch = torch_cuda
    from paper_2103_15418_b200.binding import HostResult
    s, p, lpf = _make(2, torch)
    pipe = O.OraclePipeline(p, s.mask, direct=False)
    res = HostResult(p)
    for t in range(3):
        cube = s.frame(t)
        h = torch.from_numpy(cube).pin_memory()
        lpf.process_frame_host(h, t, res)
        o = pipe.step(cube, t)
        assert np.array_equal(res.band_ok.numpy(), o["band_ok"])
        assert np.array_equal(res.upos[:res.nu].numpy(), o["upos"])
        assert np.array_equal(res.cand_idx[:res.nu].numpy(), o["cand_idx"])
        assert np.array_equal(res.act_slots[:res.npos].numpy(), o["act_slots"])
        assert np.array_equal(res.flux[:res.npos].numpy(), o["flux"])
    lpf.close()


def test_fused_kernel_special_paths(torch_cuda):
    """The fused sweep's rare paths: (a) a cube that is not an exact zero at invalid pixels (the kernel then
    applies W itself), (b) more eq.-5 hits in a row pair than the candidate queue holds (tested in place),
    (c) a cube that is not 16-byte aligned (bulk copies impossible: the general path serves the call)."""
    torch = torch_cuda
    from paper_2103_15418_b200.binding import LPF
    rng = np.random.default_rng(5)
    B, D = 4, 256
    p = synth.default_params(2); p.update(B=B, Dy=D, Dx=D)
    yy, xx = np.mgrid[0:D, 0:D]
    c = (D - 1) / 2
    W = (((yy - c) ** 2 + (xx - c) ** 2) <= (0.45 * D) ** 2).astype(np.uint8)
    W[100:104, 60:90] = 0                       # a hole as well
    base = rng.standard_normal((B, D, D)).astype(np.float32)
    for (y, x, a) in [(80, 70, 12.0), (128, 128, 30.0), (150, 200, 9.0), (101, 58, 15.0), (30, 128, 10.0)]:
        g = np.exp(-0.5 * ((yy - y) ** 2 + (xx - x) ** 2) / 0.85 ** 2).astype(np.float32)
        base += a * g
    lpf = LPF(p, W)
    assert lpf.plan()["fused"]
    pipe = O.OraclePipeline(p, W, direct=False)
    # (a) garbage (also non-finite) at the invalid pixels of some frames; clean frames in between
    for t in range(4):
        cube = base + 0.1 * rng.standard_normal(base.shape).astype(np.float32)
        if t in (1, 3):
            junk = (50.0 * rng.standard_normal(base.shape)).astype(np.float32)
            cube = np.where(W[None] != 0, cube, junk)
            cube[0, 0, 0] = np.nan; cube[2, 101, 70] = np.inf
        else:
            cube = cube * W
        o = pipe.step(cube, t)
        lpf.process_frame(torch.from_numpy(cube).cuda(), t)
        gv = lpf.frame_view(0)
        r = parity.check_frame(gv, o, pipe, cube, f"dirty t={t}")
        assert r["in_sync"] and gv["band_ok"].all() and gv["upos"].size >= 4
    lpf.close()
    # (b) kappa = 1: about 80 noise pixels pass eq. 5 in every row pair of a strip (the queue holds 64), plus rows of
    # bright sources
    p2 = dict(p); p2["max_det"] = 65536; p2["kappa"] = 1.0
    W1 = np.ones((D, D), np.uint8)
    cube = rng.standard_normal((B, D, D)).astype(np.float32)
    for y in (60, 61, 130, 200):
        for x in range(8, D - 8, 5):
            g = np.exp(-0.5 * ((yy - y) ** 2 + (xx - x) ** 2) / 0.85 ** 2).astype(np.float32)
            cube += (40.0 + (x % 7)) * g
    lpf = LPF(p2, W1)
    pipe = O.OraclePipeline(p2, W1, direct=False)
    o = pipe.step(cube, 0)
    lpf.process_frame(torch.from_numpy(cube).cuda(), 0)
    gv = lpf.frame_view(0)
    assert parity.check_frame(gv, o, pipe, cube, "queue overflow")["in_sync"]
    assert gv["ndets"] > 2000 and lpf.counters()["dropped_records"] == 0
    # (c) the same frame from a pointer that is only 4-byte aligned
    big = torch.empty(cube.size + 1, dtype=torch.float32, device="cuda")
    mis = big[1:].view(B, D, D)
    mis.copy_(torch.from_numpy(cube))
    assert mis.data_ptr() % 16 != 0
    pipe2 = O.OraclePipeline(p2, W1, direct=False)
    o2 = pipe2.step(cube, 0)
    lpf2 = LPF(p2, W1)
    lpf2.process_frame(mis, 0)
    assert parity.check_frame(lpf2.frame_view(0), o2, pipe2, cube, "misaligned cube")["in_sync"]
    lpf.close(); lpf2.close()


def test_fused_very_bright_sources(torch_cuda):
    """Sources at 1e3 and 1e4 sigma (A-team sources in real AARTFAAC images) in the fused sweep: its float32 running
    sums must not keep the rounding they made while such a value was inside the window (the kernel rebuilds a sum
    from its ring when a value far above the noise leaves it), so C, S and the detections BELOW and BESIDE the bright
    sources still meet the float64 oracle within the tolerance."""
    torch = torch_cuda
    from paper_2103_15418_b200.binding import LPF
    rng = np.random.default_rng(77)
    B, D = 4, 384
    p = synth.default_params(2); p.update(B=B, Dy=D, Dx=D)
    yy, xx = np.mgrid[0:D, 0:D]

    def src(y, x, a):
        return (a * np.exp(-0.5 * ((yy - y) ** 2 + (xx - x) ** 2) / 0.85 ** 2)).astype(np.float32)

    base = np.zeros((D, D), np.float32)
    base += src(90, 100, 1.0e3) + src(200, 250, 1.0e4) + src(60, 300, 3.0e3)
    # ordinary sources where a left-over of the bright ones would show: in the rows after they leave the 25-row
    # windows, in their columns and a little beside them, and far away
    for (y, x, a) in [(118, 100, 9.0), (131, 104, 12.0), (150, 92, 8.0), (229, 250, 10.0), (245, 262, 14.0), (262, 236, 9.0),
                      (300, 250, 7.0), (90, 140, 11.0), (200, 290, 9.0), (95, 300, 8.0), (330, 60, 10.0), (20, 20, 12.0)]:
        base += src(y, x, a)
    lpf = LPF(p, None)
    assert lpf.plan()["fused"]
    pipe = O.OraclePipeline(p, None, direct=False)
    for t in range(2):
        cube = (base[None] + rng.standard_normal((B, D, D))).astype(np.float32)
        o = pipe.step(cube, t)
        lpf.process_frame(torch.from_numpy(cube).cuda(), t)
        g = lpf.frame_view(0)
        r = parity.check_frame(g, o, pipe, cube, f"bright t={t}")
        assert r["in_sync"] and g["upos"].size >= 12
    lpf.close()


def test_host_entry_point_pipelined(torch_cuda):
    """lpf_process_frame_host_begin/_end with three lanes in flight gives what the synchronous call gives."""
    torch = torch_cuda
    from paper_2103_15418_b200.binding import HostResult
    s, p, lpf = _make(2, torch, n_lanes=3)
    pipe = O.OraclePipeline(p, s.mask, direct=False)
    L = 3
    res = [HostResult(p) for _ in range(L)]
    streams = [torch.cuda.Stream() for _ in range(L)]
    cubes = [s.frame(t) for t in range(7)]
    pinned = [torch.from_numpy(c).pin_memory() for c in cubes]
    outs = []
    for t in range(7):
        ln = t % L
        if t >= L:
            lpf.process_frame_host_end(res[ln], lane=ln, stream=streams[ln])
            outs.append({k: getattr(res[ln], k)[: (res[ln].nu if k in ("upos", "cand_idx") else res[ln].npos)].numpy().copy()
                         for k in ("upos", "cand_idx", "act_slots", "flux")} | {"band_ok": res[ln].band_ok.numpy().copy()})
        lpf.process_frame_host_begin(pinned[t], t, res[ln], lane=ln, stream=streams[ln])
    for t in range(7 - L, 7):
        ln = t % L
        lpf.process_frame_host_end(res[ln], lane=ln, stream=streams[ln])
        outs.append({k: getattr(res[ln], k)[: (res[ln].nu if k in ("upos", "cand_idx") else res[ln].npos)].numpy().copy()
                     for k in ("upos", "cand_idx", "act_slots", "flux")} | {"band_ok": res[ln].band_ok.numpy().copy()})
    for t in range(7):
        o = pipe.step(cubes[t], t)
        for k in ("band_ok", "upos", "cand_idx", "act_slots", "flux"):
            assert np.array_equal(outs[t][k], o[k]), (t, k)
    lpf.close()


def test_config3_bench_launch_configuration(torch_cuda):
    """Config 3 in the configuration bench.py times: eight lanes in flight on eight streams (the plan then gives
    a fused launch a quarter of the SMs: two row segments per plane).  Frame 0 against the oracle, element by
    element; every frame against a one-lane context (eight segments per plane) fed in sequence: the two launch
    plans and the cross-lane ordering of the association chain must not change a single result."""
    torch = torch_cuda
    from paper_2103_15418_b200.binding import LPF
    s = synth.CubeStream(3)
    p = synth.default_params(3); p["n_lanes"] = 8
    lpf = LPF(p, s.mask)
    plan8 = lpf.plan()
    assert plan8["fused"] and plan8["ctas_per_plane"] == 2, plan8
    n = 8
    cubes = [s.frame(t) for t in range(n)]
    dcubes = [torch.from_numpy(c).cuda() for c in cubes]
    streams = [torch.cuda.Stream() for _ in range(n)]
    torch.cuda.synchronize()
    for t in range(n):
        lpf.process_frame(dcubes[t], t, lane=t, stream=streams[t])
    torch.cuda.synchronize()
    views = [lpf.frame_view(t) for t in range(n)]
    pipe = O.OraclePipeline(p, s.mask, direct=False)
    o0 = pipe.step(cubes[0], 0)
    assert parity.check_frame(views[0], o0, pipe, cubes[0], "cfg3 8 lanes t=0")["in_sync"]
    p1 = dict(p); p1["n_lanes"] = 1
    seq = LPF(p1, s.mask)
    assert seq.plan()["ctas_per_plane"] > 2
    for t in range(n):
        seq.process_frame(dcubes[t], t)
        v = seq.frame_view(0)
        for k in ("band_ok", "upos", "uplane", "cand_idx", "act_slots", "act_pix", "flux"):
            assert np.array_equal(v[k], views[t][k]), (t, k)
        assert v["ndets"] == views[t]["ndets"]
        a = np.sort(v["rec"], order=["plane", "pix"]); b = np.sort(views[t]["rec"], order=["plane", "pix"])
        assert np.array_equal(a["pix"], b["pix"]) and np.array_equal(a["plane"], b["plane"])
        # the running sums of the two plans start at different rows: values agree within the north_star tolerance
        assert np.allclose(a["snr"], b["snr"], rtol=1e-4, atol=1e-5) and np.allclose(a["f"], b["f"], rtol=1e-4, atol=1e-5)
        # the QC grids of the two plans differ (lpf_qs_blocks: fewer, longer blocks with lanes in flight), hence the
        # grouping of the float64 partial sums: the statistics agree within the QC tolerances, not bit for bit
        n_t = len(parity.TIES)
        parity.check_qc(v["stats"], v["band_ok"], views[t]["stats"].astype(np.float64), views[t]["band_ok"],
                        f"cfg3 1 lane vs 8 lanes t={t}", cube=cubes[t], W=s.mask, qc_clip=p["qc_clip"])
        del parity.TIES[n_t:]          # GPU against GPU: not an oracle tie
    seq.close(); lpf.close()


@pytest.mark.parametrize("T_ring,n_back", [(128, 8), (6, 12)])
def test_backward_fill(torch_cuda, T_ring, n_back):
    """O11: slots created at t are back-filled from the device cache of the last n_back cubes.
    Every active slot's dynamic spectrum must equal the oracle's bit for bit, including the pre-birth columns,
    with a rejected band in one cached frame and with a ring shorter than the cache."""
    torch = torch_cuda
    s, p, lpf = _make(2, torch, T_ring=T_ring, n_back=n_back)
    pipe = O.OraclePipeline(p, s.mask, direct=False)
    n = 26
    for t in range(n):
        cube = s.frame(t)
        if t == 9:
            cube = cube.copy(); cube[3, 5, 5] = np.nan          # band 3 rejected in this frame
        o = pipe.step(cube, t)
        lpf.process_frame(torch.from_numpy(cube).cuda(), t)
        g = lpf.frame_view(0)
        assert np.array_equal(g["band_ok"], o["band_ok"]) and np.array_equal(g["upos"], o["upos"])
        assert np.array_equal(g["cand_idx"], o["cand_idx"]) and np.array_equal(g["act_slots"], o["act_slots"])
    tb = pipe.table
    act = np.flatnonzero(tb.active)
    late = [int(sl) for sl in act if tb.born[sl] > 2]            # born late enough to have something to back-fill
    assert len(late) >= 2
    n_pre = 0
    for sl in act:
        a = lpf.get_dynspec(int(sl), n - 1).cpu().numpy(); b = tb.dynspec(int(sl), n - 1)
        assert np.array_equal(np.isnan(a), np.isnan(b)), int(sl)
        assert np.array_equal(a[~np.isnan(a)], b[~np.isnan(b)]), int(sl)
        if tb.born[sl] > 2:
            k = T_ring - 1 - (n - 1 - int(tb.born[sl]))         # column of the birth frame (newest frame is last)
            if k >= 1:
                n_pre += int(not np.isnan(b[:, k - 1]).any())
    assert n_pre >= 1                                             # the build-up columns are really there
    lpf.close()


def test_backward_fill_with_lanes_in_flight(torch_cuda):
    """O11 with four frames in flight: the cache holds n_back + n_lanes cubes, so a lane's early copy into the
    cache never overwrites a cube that a frame still in flight on another lane back-fills from."""
    torch = torch_cuda
    L, n_back, n = 4, 3, 24
    s, p, lpf = _make(2, torch, T_ring=32, n_back=n_back, n_lanes=L)
    pipe = O.OraclePipeline(p, s.mask, direct=False)
    streams = [torch.cuda.Stream() for _ in range(L)]
    cubes = [s.frame(t) for t in range(n)]
    dcubes = [torch.from_numpy(c).cuda() for c in cubes]
    torch.cuda.synchronize()
    for t0 in range(0, n, L):
        for k in range(L):
            lpf.process_frame(dcubes[t0 + k], t0 + k, lane=k, stream=streams[k])
        torch.cuda.synchronize()
        for k in range(L):
            o = pipe.step(cubes[t0 + k], t0 + k)
            g = lpf.frame_view(k)
            assert np.array_equal(g["upos"], o["upos"]) and np.array_equal(g["cand_idx"], o["cand_idx"])
            assert np.array_equal(g["act_slots"], o["act_slots"]) and np.array_equal(g["flux"], o["flux"])
    tb = pipe.table
    for sl in np.flatnonzero(tb.active):
        a = lpf.get_dynspec(int(sl), n - 1).cpu().numpy(); b = tb.dynspec(int(sl), n - 1)
        assert np.array_equal(np.isnan(a), np.isnan(b)), int(sl)
        assert np.array_equal(a[~np.isnan(a)], b[~np.isnan(b)]), int(sl)
    lpf.close()


def test_checkpoint_resume(torch_cuda):
    """lpf_export_state / lpf_import_state: a second context that imports the blob written after
    frame 13 continues the stream bit for bit - against the context that never stopped AND against the oracle that
    ran all frames (candidate table, rings incl. the backward fill from the cached cubes, eq. A.2 running state).
    A blob from a context with other parameters is refused."""
    torch = torch_cuda
    from paper_2103_15418_b200.binding import LPF, LpfError
    kw = dict(T_ring=16, n_back=3, zeta_thr=12.0, zeta_nmax=3, zeta_window=16, zeta_warm=8)
    s, p, lpf_a = _make(2, torch, **kw)
    pipe = O.OraclePipeline(p, s.mask, direct=False)
    n0, n1 = 14, 24
    outs = []
    for t in range(n0):
        outs.append(pipe.step(s.frame(t), t))
        lpf_a.process_frame(torch.from_numpy(s.frame(t)).cuda(), t)
    blob = lpf_a.export_state()
    assert blob.nbytes == lpf_a.lib.lpf_state_bytes(lpf_a.h) and bytes(blob[:8]) == b"LPFSTATE"
    lpf_b = LPF(p, s.mask)
    lpf_b.import_state(blob)
    other = dict(p); other["n_forget"] = p["n_forget"] + 1
    lpf_c = LPF(other, s.mask)
    with pytest.raises(LpfError):
        lpf_c.import_state(blob)
    with pytest.raises(LpfError):
        lpf_b.import_state(blob[:-8])
    lpf_c.close()
    keys = ("band_ok", "upos", "uplane", "cand_idx", "act_slots", "act_pix", "flux")
    for t in range(n0, n1):
        cube = s.frame(t)
        o = pipe.step(cube, t)
        d = torch.from_numpy(cube).cuda()
        lpf_a.process_frame(d, t); lpf_b.process_frame(d, t)
        ga, gb = lpf_a.frame_view(0), lpf_b.frame_view(0)
        for k in keys:
            assert np.array_equal(ga[k], gb[k], equal_nan=True), (t, k)
        assert np.array_equal(gb["upos"], o["upos"]) and np.array_equal(gb["cand_idx"], o["cand_idx"])
        assert np.array_equal(gb["act_slots"], o["act_slots"]) and np.array_equal(gb["flux"], o["flux"])
    tb = pipe.table
    act = np.flatnonzero(tb.active)
    assert act.size > 10 and any(n0 <= tb.born[sl] < n0 + 3 for sl in act)      # slots back-filled from imported cubes
    for sl in act:
        a = lpf_a.get_dynspec(int(sl), n1 - 1).cpu().numpy(); b = lpf_b.get_dynspec(int(sl), n1 - 1).cpu().numpy()
        ob = tb.dynspec(int(sl), n1 - 1)
        assert np.array_equal(a, b, equal_nan=True), int(sl)
        assert np.array_equal(np.isnan(b), np.isnan(ob)) and np.array_equal(b[~np.isnan(b)], ob[~np.isnan(ob)]), int(sl)
    assert lpf_a.counters()["n_active"] == lpf_b.counters()["n_active"] == act.size
    lpf_a.close(); lpf_b.close()


def test_running_pixel_qc(torch_cuda):
    """O12 (eq. A.2): per-pixel running mean / variance, test before update, update only accepted
    bands.  The oracle evaluates eq. A.2 in float64 on its float32 state; the per-band counts of the kernel (plain
    float32) may differ from the oracle's only by pixels whose ORACLE margin |d^2 - thr^2 v| is within 2e-4 relative
    (oracle's `near` count; every such difference is logged as a tie), the band verdicts must be equal; the rest of
    the chain follows band_ok.  Also: the start-over rule (zeta_reset) after a lasting level change."""
    torch = torch_cuda
    s, p, lpf = _make(2, torch, zeta_thr=12.0, zeta_nmax=3, zeta_window=16, zeta_warm=8, n_lanes=2)
    pipe = O.OraclePipeline(p, s.mask, direct=False)
    rng = np.random.default_rng(4)
    streams = [torch.cuda.Stream() for _ in range(2)]
    n_rej = 0
    for t in range(24):
        cube = s.frame(t)
        if t in (12, 13, 19):                              # short-lived local interference in one or two bands
            cube = cube.copy()
            for b in ((5,) if t != 13 else (5, 9)):
                for _ in range(6):
                    cube[b, rng.integers(10, 240), rng.integers(10, 240)] += 400.0
        o = pipe.step(cube, t)
        lpf.process_frame(torch.from_numpy(cube).cuda(), t, lane=t % 2, stream=streams[t % 2])
        g = lpf.frame_view(t % 2)
        dz = np.abs(g["zeta_cnt"].astype(np.int64) - o["zeta_cnt"])
        assert np.all(dz <= o["zeta_near"]), (t, g["zeta_cnt"], o["zeta_cnt"], o["zeta_near"])
        for b in np.flatnonzero(dz):
            parity.TIES.append((f"running qc t={t}", int(b), -1, "zeta", float(dz[b])))
        assert np.array_equal(g["band_ok"], o["band_ok"]), t
        r = parity.check_frame(g, o, pipe, cube, f"running qc t={t}")
        assert r["in_sync"]
        n_rej += int((o["band_ok"][:-1] == 0).sum())
        if t in (12, 13, 19):
            assert o["band_ok"][5] == 0 and o["zeta_cnt"][5] >= 6
    assert n_rej >= 4
    lpf.close()
    # a lasting local level change in one band (a 3x3 patch 14 sigma brighter from t = 16 on; small enough to pass
    # eq. A.1): discarded three frames in a row, then the band starts over, is untested during its new warm-up and
    # comes back for good
    s, p, lpf = _make(2, torch, zeta_thr=10.0, zeta_nmax=3, zeta_window=16, zeta_warm=12, zeta_reset=3)
    pipe = O.OraclePipeline(p, s.mask, direct=False)
    seen = []
    for t in range(36):
        cube = s.frame(t)
        if t >= 16:
            cube = cube.copy(); cube[7, 100:103, 60:63] += 14.0
        o = pipe.step(cube, t)
        lpf.process_frame(torch.from_numpy(cube).cuda(), t)
        g = lpf.frame_view(0)
        assert np.all(np.abs(g["zeta_cnt"].astype(np.int64) - o["zeta_cnt"]) <= o["zeta_near"]), t
        assert np.array_equal(g["band_ok"], o["band_ok"]), t
        seen.append(int(g["band_ok"][7]))
    assert seen[:16] == [1] * 16 and seen[16:19] == [0, 0, 0] and seen[19:] == [1] * 17, seen
    lpf.close()


def test_network_input_export_and_pulse_simulator(torch_cuda):
    """O13 (batched, ordered, sigma-normalised dynamic spectra, bit-exact) and O14 (eqs. 19-21 pulses,
    float32 kernel against the float64 oracle) and their combination (injection into exported spectra)."""
    torch = torch_cuda
    from paper_2103_15418_b200.binding import simulate_pulses
    s, p, lpf = _make(2, torch, T_ring=24)
    pipe = O.OraclePipeline(p, s.mask, direct=False)
    n = 30
    for t in range(n):
        cube = s.frame(t)
        o = pipe.step(cube, t)
        lpf.process_frame(torch.from_numpy(cube).cuda(), t)
    g = lpf.frame_view(0)
    assert np.array_equal(g["act_slots"], o["act_slots"])
    slots = o["act_slots"][::3].astype(np.int32)
    sigma = g["stats"][:, 5].astype(np.float32)               # clipped rms per band
    for t_last, sg in ((n - 1, sigma), (n + 4, None)):
        x = lpf.export_dynspec(torch.from_numpy(slots).cuda(), t_last, None if sg is None else torch.from_numpy(sg).cuda())
        ref = O.export_dynspec(pipe.table, slots, t_last, sg)
        assert x.shape == ref.shape and np.array_equal(x.cpu().numpy(), ref)
        assert not np.isnan(ref).any()
    # simulator
    rng = np.random.default_rng(8)
    B, T = p["B"], 24
    nu = np.array(s.c.nu_mhz if hasattr(s.c, "nu_mhz") else np.linspace(57.0, 63.1, B), np.float32)
    nu0 = float(nu.max())
    m = slots.size
    theta = np.stack([rng.uniform(2, T - 2, m), rng.uniform(0.8, 6, m), rng.uniform(0, 40, m), rng.uniform(0, 8, m),
                      rng.uniform(-4, 4, m)], 1).astype(np.float32)
    I = simulate_pulses(torch.from_numpy(theta).cuda(), torch.from_numpy(nu).cuda(), nu0, T, dt_s=1.0).cpu().numpy()
    ref = O.simulate_pulses(theta.astype(np.float64), nu.astype(np.float64), nu0, T, 1.0)
    assert np.allclose(I, ref, rtol=2e-4, atol=2e-5 * float(theta[:, 3].max()))
    # injection into the exported spectra (accumulate)
    x = lpf.export_dynspec(torch.from_numpy(slots).cuda(), n - 1, torch.from_numpy(sigma).cuda())
    x0 = x.cpu().numpy().copy()
    simulate_pulses(torch.from_numpy(theta).cuda(), torch.from_numpy(nu).cuda(), nu0, T, 1.0, out=x, accumulate=True)
    assert np.allclose(x.cpu().numpy(), x0 + ref, rtol=2e-4, atol=1e-4)
    lpf.close()
