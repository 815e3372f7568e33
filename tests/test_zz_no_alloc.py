"""far_voxelize_static -- the entry point for callers that cannot allocate device memory -- against far_voxelize.

Some users of this library are not in a position to call cudaMalloc: a LiDAR callback inside a real-time loop (the
call takes driver-wide locks and may synchronise the device for as long as it likes), or a component that runs on
buffers handed to it by a host application that owns the GPU memory budget.  far_voxelize_static serves them from a
fixed scratch array inside libfar.so (FAR_VOXELIZE_STATIC_BYTES per GPU, scans of at most
FAR_VOXELIZE_STATIC_MAX_POINTS points).  All calls share that array and it keeps the previous call's contents, so the
test makes TWO calls in a row on different scans -- the second one starts on a dirty scratch -- and wants each to equal
what the existing path (far_voxelize with a caller workspace) returns for the same scan.  Voxelisation is index work:
the tolerance is the one the other voxelise tests use, bit equality of indices and coordinates.

The file is named so that pytest collects it last: `pytest -x` stops at the first failure, and a failure here must
not hide the parity tests.  It passes both alone in a fresh process (the first call does the per-device address
look-up) and after the rest of the suite (other tests have then used the GPU and the library already)."""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu

far = pytest.importorskip("paper_2606_26010_b200")


def _scan(seed, n, scale):
    """uniform points plus a dense blob (many points per voxel) and two non-finite rows the voxeliser must skip"""
    rng = np.random.default_rng(seed)
    pts = rng.uniform(-scale, scale, size=(n, 3))
    pts[: n // 3] = rng.normal(0.0, 0.6, size=(n // 3, 3)) + np.array([3.0, -2.0, 1.0])
    pts = pts.astype(np.float32)
    if n > 10:
        pts[3] = np.nan
        pts[n // 2] = np.inf
    return pts


def _static(x, voxel, out_xyz, out_index, n_out, poison):
    """one far_voxelize_static call into caller-owned buffers; nothing is allocated between the calls under test"""
    out_xyz.fill_(poison)
    out_index.fill_(-7)
    n_out.fill_(-1)
    far.voxelize_static(x, voxel, out_xyz, out_index, n_out)
    m = int(n_out.item())
    return out_xyz[:m].cpu().numpy(), out_index[:m].cpu().numpy()


def test_static_scratch_voxelize_equals_workspace_path_on_two_calls_in_a_row():
    n_max = far.VOXELIZE_STATIC_MAX_POINTS
    # call 1: a full-size scan (every byte of the scratch gets used); call 2: a smaller, ragged one at another voxel size,
    # whose hash table lands on the slots call 1 dirtied; call 3: the empty scan
    cases = [(_scan(101, n_max, 60.0), 0.5), (_scan(202, 77_777, 40.0), 1.0), (np.zeros((0, 3), np.float32), 1.0)]
    dev = [torch.as_tensor(p).cuda() for p, _ in cases]
    # expected values from the existing path, taken BEFORE the calls under test so that nothing runs in between them
    want = [far.Voxelizer(max(len(p), 1))(x, v) for (p, v), x in zip(cases, dev)]
    want = [(a.cpu().numpy(), b.cpu().numpy()) for a, b in want]
    assert len(want[0][1]) > 1000 and len(want[1][1]) > 1000 and len(want[2][1]) == 0

    out_xyz = torch.empty((n_max, 3), dtype=torch.float32, device="cuda")
    out_index = torch.empty(n_max, dtype=torch.int32, device="cuda")
    n_out = torch.empty(1, dtype=torch.int64, device="cuda")
    torch.cuda.synchronize()
    launches = far.launch_count()
    got = [_static(x, v, out_xyz, out_index, n_out, poison) for x, (_, v), poison in zip(dev, cases, (1e30, -1e30, 0.0))]
    assert far.launch_count() == launches + 4 + 4 + 1          # the library's own kernels ran: 4 per scan, 1 for n = 0
    for (g_xyz, g_idx), (w_xyz, w_idx) in zip(got, want):
        assert np.array_equal(g_idx, w_idx)
        assert np.array_equal(g_xyz.view(np.uint32), w_xyz.view(np.uint32))

    # and once more in the opposite order: big after small, again on whatever the last call left behind
    g_xyz, g_idx = _static(dev[0], cases[0][1], out_xyz, out_index, n_out, 5.0)
    assert np.array_equal(g_idx, want[0][1]) and np.array_equal(g_xyz.view(np.uint32), want[0][0].view(np.uint32))


def test_static_scratch_voxelize_refuses_scans_beyond_its_limit():
    n = far.VOXELIZE_STATIC_MAX_POINTS + 1
    x = torch.zeros((n, 3), dtype=torch.float32, device="cuda")
    out_xyz = torch.full((n, 3), 3.0, dtype=torch.float32, device="cuda")
    out_index = torch.full((n,), -7, dtype=torch.int32, device="cuda")
    n_out = torch.full((1,), -1, dtype=torch.int64, device="cuda")
    with pytest.raises(far.FarError) as e:
        far.voxelize_static(x, 1.0, out_xyz, out_index, n_out)
    assert e.value.status == far.ERR_ARG
    assert b"FAR_VOXELIZE_STATIC_MAX_POINTS (262144)" in far.lib().far_last_cuda_error()
    torch.cuda.synchronize()
    assert int(n_out.item()) == -1 and int(out_index[0].item()) == -7      # refused before anything was enqueued
