"""-m gpu, collected last: lpf_cube_qc_static, the entry point that allocates nothing (its scratch is a static device
array inside the library), against the existing lpf_cube_qc on the same cubes, within the QC tolerances of
tests/parity.py (check_qc: n and band_ok exact, moments within the north_star tolerance, clip-boundary pixels
classified from the cube).  Passes alone in a fresh process and after the other tests: it builds its own contexts
and leaves nothing behind but the shared static array, which every call re-initialises."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_2103_15418_b200 import synth
import parity


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available()
    return torch


def _same_as_lane_path(lpf, s, p, d_cube, h_cube, stats_buf, ok_buf, tag):
    """One static call into caller-owned outputs vs one lpf_cube_qc call on the same cube."""
    torch = lpf.torch
    st_l, ok_l = lpf.cube_qc(d_cube)
    lpf.cube_qc_static(d_cube, stats=stats_buf, ok=ok_buf)
    torch.cuda.synchronize()
    n_before = len(parity.TIES)
    parity.check_qc(stats_buf.cpu().numpy(), ok_buf.cpu().numpy(), st_l.cpu().numpy().astype(np.float64), ok_l.cpu().numpy(),
                    tag, cube=h_cube, W=s.mask, qc_clip=p["qc_clip"])
    del parity.TIES[n_before:]          # GPU-vs-GPU boundary pixels are not oracle ties: keep them out of the tie log
    return ok_l.cpu().numpy()


def test_static_scratch_qc_matches_lane_qc(torch_cuda):
    torch = torch_cuda
    from paper_2103_15418_b200.binding import LPF
    s = synth.CubeStream(2)
    p = synth.default_params(2)
    lpf = LPF(p, s.mask)
    B = p["B"]
    stats_buf = torch.empty((B, 8), dtype=torch.float32, device="cuda")
    ok_buf = torch.empty((B + 1,), dtype=torch.uint8, device="cuda")
    # frame A: clean; frame B: two bands with interference (rejected by eq. A.1) and a NaN in a third
    cube_a = s.frame(0)
    cube_b = s.frame(1).copy()
    cube_b[3] = cube_b[3] * 9.0 + 4.0
    cube_b[7] += 2.5
    cube_b[11, 100, 100] = np.nan
    d_a, d_b = torch.from_numpy(cube_a).cuda(), torch.from_numpy(cube_b).cuda()
    _same_as_lane_path(lpf, s, p, d_a, cube_a, stats_buf, ok_buf, "static warm-up")   # set-up call (symbol address)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    # two calls in a row on different cubes, then the first cube again: the array keeps the last call's contents
    ok_a = _same_as_lane_path(lpf, s, p, d_a, cube_a, stats_buf, ok_buf, "static A")
    ok_b = _same_as_lane_path(lpf, s, p, d_b, cube_b, stats_buf, ok_buf, "static B")
    ok_a2 = _same_as_lane_path(lpf, s, p, d_a, cube_a, stats_buf, ok_buf, "static A again")
    assert ok_a.all() and np.array_equal(ok_a, ok_a2)
    assert ok_b[3] == 0 and ok_b[7] == 0 and ok_b[11] == 0 and ok_b[B] == 1 and ok_b.sum() == B + 1 - 3
    # back to back on one stream without a synchronise in between: the second call's result is the one that stays
    lpf.cube_qc_static(d_b, stats=stats_buf, ok=ok_buf)
    lpf.cube_qc_static(d_a, stats=stats_buf, ok=ok_buf)
    torch.cuda.synchronize()
    assert np.array_equal(ok_buf.cpu().numpy(), ok_a)
    assert torch.cuda.mem_get_info()[0] == free0          # the device's free memory did not move: nothing was allocated
    # a cube that is not 16-byte aligned (both sides take the generic kernels)
    big = torch.empty(cube_a.size + 1, dtype=torch.float32, device="cuda")
    mis = big[1:].view(cube_a.shape)
    mis.copy_(d_b)
    assert mis.data_ptr() % 16 != 0
    _same_as_lane_path(lpf, s, p, mis, cube_b, stats_buf, ok_buf, "static misaligned")
    lpf.close()


def test_static_scratch_qc_on_the_headline_shape_and_its_limit(torch_cuda):
    torch = torch_cuda
    from paper_2103_15418_b200.binding import LPF, LpfError, E_TOO_LARGE
    # config 3 (1024 x 1024 x 16), one frame with an RFI band
    s = synth.CubeStream(3)
    p = synth.default_params(3)
    lpf = LPF(p, s.mask)
    cube = s.frame(0).copy()
    cube[5] *= 3.0
    d = torch.from_numpy(cube).cuda()
    stats_buf = torch.empty((p["B"], 8), dtype=torch.float32, device="cuda")
    ok_buf = torch.empty((p["B"] + 1,), dtype=torch.uint8, device="cuda")
    for k in range(2):
        ok = _same_as_lane_path(lpf, s, p, d, cube, stats_buf, ok_buf, f"static cfg3 call {k}")
        assert ok[5] == 0 and ok.sum() == p["B"]
    lpf.close()
    # beyond the static array: 64 bands x (64 + 640) blocks x 24 bytes > 1 MiB -> refused, nothing launched
    big = synth.default_params(3)
    big.update(B=64, Dy=1280, Dx=1024, n_cand_max=64, T_ring=4, n_lanes=1)
    lpf = LPF(big, None)
    dummy = torch.zeros(16, dtype=torch.float32, device="cuda")
    stats_buf = torch.full((64, 8), -7.0, dtype=torch.float32, device="cuda")
    ok_buf = torch.full((65,), 9, dtype=torch.uint8, device="cuda")
    with pytest.raises(LpfError) as ei:
        lpf.cube_qc_static(dummy, stats=stats_buf, ok=ok_buf)
    assert f"({E_TOO_LARGE})" in str(ei.value) and "LPF_QC_STATIC_BYTES" in str(ei.value)
    torch.cuda.synchronize()
    assert bool((stats_buf == -7.0).all()) and bool((ok_buf == 9).all())
    lpf.close()
