"""GPU parity for the SURVEY 8(f) rows: motion undistortion (R15/R16) and Adaptive Submap Density
(R17) -- CUDA path through the C ABI vs the FP64 CPU oracle on the same seeded inputs.

Tolerances: ASMD decides integers (limits, contents, ids, counts) -> bit-exact.  Undistortion
is FP64 on both sides with a different but equivalent evaluation order (series vs libm sin/cos, cross products vs
matrix) -> results agree to ~1e-15 relative before the single rounding to fp32, so outputs are identical except
where that tiny difference straddles an fp32 rounding boundary: at most 1 ulp, on a vanishing fraction of values.
"""
import math

import numpy as np
import pytest
import torch

import far_scenes as scenes
import oracle

pytestmark = pytest.mark.gpu

far = pytest.importorskip("paper_2606_26010_b200")


def _ulp_diff(a, b):
    ia = a.view(np.int32).astype(np.int64)
    ib = b.view(np.int32).astype(np.int64)
    ia = np.where(ia < 0, -(ia & 0x7FFFFFFF), ia)
    ib = np.where(ib < 0, -(ib & 0x7FFFFFFF), ib)
    return np.abs(ia - ib)


def _assert_undistort_parity(g, o):
    assert g.shape == o.shape
    d = _ulp_diff(np.ascontiguousarray(g), np.ascontiguousarray(o))
    assert d.max() <= 1, d.max()
    assert (d > 0).mean() <= 1e-4, (d > 0).mean()


# ---- undistortion ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n", [0, 1, 5, 1023, 1024, 1025, 4099, 100_003])
@pytest.mark.parametrize("stride", [3, 4])
def test_undistort_matches_oracle_sizes_and_strides(n, stride):
    rng = np.random.default_rng(n + stride)
    p = rng.uniform(-150, 150, (n, stride)).astype(np.float32)
    t = rng.uniform(0, 0.1, n).astype(np.float32)
    a = np.array([69.4, 0.3, -0.1, 0.01, -0.02, 0.25])
    b = np.array([-4.0, 0.5, 0.0, 0.0, 0.0, 0.6])
    o = oracle.undistort(p, t, 0.1, a, b) if n else np.zeros((0, 3), np.float32)
    if n == 0:
        g = far.undistort(torch.zeros((0, stride), device="cuda"), torch.zeros(0, device="cuda"), 0.1, a, b)
        assert g.shape == (0, 3)
        return
    g = far.undistort(p, t, 0.1, a, b).cpu().numpy()
    _assert_undistort_parity(g, o)


@pytest.mark.parametrize("case", ["racing", "spinning", "aggressive", "large_angle", "zero"])
def test_undistort_motion_cases(case):
    cfg = {"racing": (dict(seed=5), 0.1),
           "spinning": (dict(seed=6, a=[12.0, 0.2, 0.0, 0.02, 0.01, 0.6], b=[1.5, 0.0, 0.0, 0.0, 0.0, -1.0]), 0.1),
           "aggressive": (dict(seed=7, a=[30.0, -5.0, 2.0, 0.5, -0.4, 1.5], b=[-20.0, 8.0, 3.0, 2.0, 1.0, -3.0]), 0.1),
           # |phi| up to 1.2 rad: beyond the series range, exercises the sincos branch
           "large_angle": (dict(seed=8, a=[5.0, 0.0, 0.0, 2.0, -4.0, 11.0], b=[0.0, 0.0, 0.0, 1.0, 0.0, 0.0], steps=400), 0.1),
           "zero": (dict(seed=9, a=np.zeros(6), b=np.zeros(6), steps=10), 0.1)}[case][0]
    d = scenes.motion_distorted_scan(n=30_000, **cfg)
    o = oracle.undistort(d["observed"], d["time"], d["dt_ref"], d["a"], d["b"])
    g = far.undistort(d["observed"], d["time"], d["dt_ref"], d["a"], d["b"]).cpu().numpy()
    _assert_undistort_parity(g, o)
    if case == "zero":
        assert np.array_equal(g.view(np.uint32), d["observed"].view(np.uint32))
    elif case != "large_angle":     # (12 rad/s is far outside the Magnus expansion's accuracy claim: parity only)
        # and the CUDA result recovers the static world like the oracle does (the oracle's pin, re-checked here)
        err = np.linalg.norm(g.astype(np.float64) - d["world"], axis=1).max()
        assert err <= (6e-5 if case == "aggressive" else 2e-5), err


def test_undistort_nonfinite_and_misaligned_views():
    rng = np.random.default_rng(3)
    p = rng.uniform(-50, 50, (5000, 3)).astype(np.float32)
    t = rng.uniform(0, 0.1, 5000).astype(np.float32)
    p[17, 0] = np.nan
    p[4000, 2] = np.inf
    t[99] = np.nan
    a, b = [20, 1, 0, 0.1, 0, 0.5], [1, 0, 0, 0, 0, 0.2]
    o = oracle.undistort(p, t, 0.1, a, b)
    g = far.undistort(p, t, 0.1, a, b).cpu().numpy()
    assert np.array_equal(g[[17, 4000, 99]].view(np.uint32), p[[17, 4000, 99]].view(np.uint32))
    keep = np.ones(5000, bool); keep[[17, 4000, 99]] = False
    _assert_undistort_parity(g[keep], o[keep])
    # input and output that are only 4-byte aligned (views offset by one point): the scalar path
    buf = torch.as_tensor(np.r_[np.zeros(3, np.float32), p.ravel()]).cuda()
    view = buf[3:].view(5000, 3)
    outbuf = torch.zeros(3 + 5000 * 3, dtype=torch.float32, device="cuda")
    out = outbuf[3:].view(5000, 3)
    far.undistort(view, t, 0.1, a, b, out=out)
    assert np.array_equal(out.cpu().numpy().view(np.uint32), g.view(np.uint32))


def test_undistort_fitted_history_chain():
    d = scenes.motion_distorted_scan(n=20_000, seed=11, history_noise=0.05)
    a, b = far.motion_fit(d["hist_times"], d["hist_vel"], d["t_ref"])
    ao, bo = oracle.motion_fit(d["hist_times"], d["hist_vel"], d["t_ref"])
    o = oracle.undistort(d["observed"], d["time"], d["dt_ref"], ao, bo)
    g = far.undistort(d["observed"], d["time"], d["dt_ref"], a, b).cpu().numpy()
    _assert_undistort_parity(g, o)


# ---- ASMD -----------------------------------------------------------------------------------------------------
def _same_contents(g, o):
    assert np.array_equal(g["keys"], o["keys"])
    assert np.array_equal(g["counts"], o["counts"])
    assert np.array_equal(g["ids"], o["ids"])
    assert np.array_equal(g["xyz"].view(np.uint32), o["xyz"].view(np.uint32))


def _planar(rng, n, half, z=0.5):
    return np.c_[rng.uniform(-half, half, (n, 2)), z + rng.normal(0, 0.02, n)].astype(np.float32)


@pytest.mark.parametrize("r_close", [0.3, 2.0, 7.5, 1e3])
def test_asmd_density_bit_exact(r_close):
    c1 = scenes.c1_tiny(seed=0)
    mo, mg = oracle.Map(0.5, 20), far.Map(0.5, 20, 1 << 13)
    mo.insert(c1["scan"]); mg.insert(c1["scan"])
    centre = [1.0, 1.0, 0.0]
    want = mo.asmd_density(centre, r_close)
    got = mg.asmd_density(centre, r_close).cpu().numpy()
    assert (float(got[0]), int(got[1])) == want


def test_asmd_density_empty_map_is_cap():
    mg = far.Map(0.5, 20, 1 << 10)
    got = mg.asmd_density([0, 0, 0], 5.0).cpu().numpy()
    assert (got[0], got[1]) == (20.0, 0.0)


@pytest.mark.parametrize("n_close,d_max", [(16.0, 80.0), (19.4, 45.0), (35.0, 1e9), (0.0, 50.0), (12.5, 30.0)])
def test_asmd_insert_contents_bit_exact(n_close, d_max):
    rng = np.random.default_rng(3)
    pts = _planar(rng, 300_000, 60.0)
    mo, mg = oracle.Map(1.0, 20), far.Map(1.0, 20, 1 << 16)
    so = mo.insert_asmd(pts, n_close, d_max)
    sg = mg.insert_asmd(pts, n_close, d_max)
    assert sg == so
    _same_contents(mg.export(), mo.export())


def test_asmd_insert_with_pose_batches_and_covariances():
    """two frames from two poses, host pose and device pose, n_close from far_asmd_density of a scan-local map;
    the second frame meets voxels that are already above their (now smaller) limit"""
    rng = np.random.default_rng(4)
    scan = _planar(rng, 80_000, 30.0)
    T1 = scenes.pose_from_rpy_t(0.0, 0.0, 0.3, [40.0, -10.0, 0.5])
    T2 = scenes.pose_from_rpy_t(0.01, -0.02, 0.35, [65.0, -10.0, 0.5])
    lo, lg = oracle.Map(1.0, 20), far.Map(1.0, 20, 1 << 14)
    lo.insert(scan); lg.insert(scan)
    n_close_o, _ = lo.asmd_density([0, 0, 0], 10.0)
    d_dens = lg.asmd_density([0, 0, 0], 10.0)
    assert float(d_dens[0].item()) == n_close_o
    mo, mg = oracle.Map(1.0, 20), far.Map(1.0, 20, 1 << 15, with_cov=True)
    so = mo.insert_asmd(scan, n_close_o, 40.0, pose=T1, compute_cov=True)
    sg = mg.insert_asmd(scan, d_dens, 40.0, pose=T1, compute_cov=True)
    assert sg == so
    d_pose = torch.as_tensor(np.frombuffer(bytes(far.Pose.from_rt(T2)), dtype=np.float64).copy()).cuda()
    so = mo.insert_asmd(scan, n_close_o, 40.0, pose=T2, compute_cov=True)
    mg.insert_asmd_enqueue(scan, d_dens, 40.0, d_pose=d_pose, compute_cov=True)
    torch.cuda.synchronize()
    sg = dict(zip(far.INSERT_STATS_FIELDS, mg._insert_stats.tolist()))
    assert sg == so
    eo, eg = mo.export(with_cov=True), mg.export(with_cov=True)
    _same_contents(eg, eo)
    assert np.array_equal(eg["cov_valid"], eo["cov_valid"])
    v = eo["cov_valid"].astype(bool)
    a, b = eg["cov"][v].astype(np.float64), eo["cov"][v].astype(np.float64)
    assert (np.linalg.norm(a - b, axis=1) / np.linalg.norm(b, axis=1)).max() < 1e-4


def test_asmd_equals_plain_insert_when_limit_is_cap():
    c1 = scenes.c1_tiny(seed=0)
    a, b = far.Map(0.5, 20, 1 << 13), far.Map(0.5, 20, 1 << 13)
    a.insert(c1["map_points"]); b.insert_asmd(c1["map_points"], 40.0, 1e9)
    _same_contents(a.export(), b.export())


def test_frontend_sweep_with_asmd_matches_oracle_chain():
    """far_frontend_process_sweep with cfg.asmd: undistort -> voxelise -> Sigma_s -> register -> density ->
    ASMD insert with covariances -> prune, against the same chain spelled out with the oracle."""
    c1 = scenes.c1_tiny(seed=0)
    v, cap = c1["voxel"], c1["cap"]
    rng = np.random.default_rng(12)
    scan = c1["scan"]
    t = np.sort(rng.uniform(0, 0.1, len(scan))).astype(np.float32)
    a_, b_ = np.array([2.0, 0.1, 0.0, 0.0, 0.0, 0.2]), np.array([0.5, 0, 0, 0, 0, 0.1])
    fe = far.Frontend(v, cap, 1 << 14, len(scan), ds_voxel=v, prune_radius=6.0, max_iters=c1["max_iters"],
                      asmd=True, asmd_r_close=3.0, asmd_d_max=12.0)
    fe.map.insert(c1["map_points"], compute_cov=True)
    mo = oracle.Map(v, cap)
    mo.insert(c1["map_points"], compute_cov=True)
    d_res = torch.zeros(far.GICP_RESULT_BYTES, dtype=torch.uint8, device="cuda")
    fe.process_sweep_enqueue(torch.as_tensor(scan).cuda(), torch.as_tensor(t).cuda(), 0.1, a_, b_, c1["T_init"], c1["sigma"],
                             d_result=d_res)
    torch.cuda.synchronize()
    g = far.result_to_dict(far.GicpResult.from_buffer_copy(d_res.cpu().numpy().tobytes()))
    # oracle chain; the undistorted sweep is taken from the CUDA path where it differs by an ulp (checked above), so
    # that the integer stages downstream see identical inputs
    und_o = oracle.undistort(scan, t, 0.1, a_, b_)
    und_g = far.undistort(scan, t, 0.1, a_, b_).cpu().numpy()
    _assert_undistort_parity(und_g, und_o)
    und = und_g
    ds, _ = oracle.voxelize(und, v)
    lo = oracle.Map(v, cap); lo.insert(und)
    cov, val = lo.knn_cov(ds)
    o = mo.gicp_register(ds, cov, val, c1["T_init"], c1["sigma"], c1["max_iters"])
    assert g["status"] == 0 and g["iters"] == o["iters"] and g["n_inliers"] == o["n_inliers"]
    assert np.linalg.norm(g["t"] - o["t"]) < 1e-4
    n_close, _ = lo.asmd_density([0, 0, 0], 3.0)
    mo.insert_asmd(und, n_close, 12.0, pose=(g["R"], g["t"]), compute_cov=True)
    mo.prune(g["t"], 6.0)
    eo, eg = mo.export(with_cov=True), fe.map.export(with_cov=True)
    _same_contents(eg, eo)
    assert np.array_equal(eg["cov_valid"], eo["cov_valid"])


# ---- R21: regular spacing -- contents bit-exact against the oracle's sequential rule ------------------------
def _spaced_cloud(rng, n):
    pts = np.concatenate([rng.uniform(-20, 20, size=(n, 3)), rng.normal(0, 0.4, size=(n // 2, 3)) + [3.0, 2.0, 1.0],
                          rng.normal(0, 0.05, size=(n // 4, 3)) + [-9.0, 7.0, 0.5]]).astype(np.float32)
    rng.shuffle(pts)
    return pts


def _same_map(g, o):
    assert np.array_equal(g["keys"], o["keys"]) and np.array_equal(g["counts"], o["counts"])
    assert np.array_equal(g["ids"], o["ids"])
    assert np.array_equal(g["xyz"].view(np.uint32), o["xyz"].view(np.uint32))


@pytest.mark.parametrize("voxel,cap,s", [(4.0, 40, 4.0 / math.sqrt(40.0)), (1.0, 20, 0.2), (2.0, 64, 0.05), (0.5, 3, 0.3)])
def test_min_spacing_insert_bit_exact(voxel, cap, s):
    rng = np.random.default_rng(50)
    pts = _spaced_cloud(rng, 60_000)
    mo = oracle.Map(voxel, cap, min_spacing=s)
    mg = far.Map(voxel, cap, 200_000, min_spacing=s, max_batch=25_000)      # calls are chunked internally
    T = scenes.pose_from_rpy_t(0.02, -0.01, 0.4, [3.0, -2.0, 0.5])
    for part, pose in ((pts[:40_000], None), (pts[40_000:90_000], T), (pts[90_000:], None)):
        assert mg.insert(part, pose=pose) == mo.insert(part, pose=pose)
    eg, eo = mg.export(), mo.export()
    _same_map(eg, eo)
    assert mg.size() == mo.size()
    # the rule's invariant on the CUDA side: no two stored points of a voxel closer than s
    for v_i in np.random.default_rng(0).choice(len(eg["keys"]), min(400, len(eg["keys"])), replace=False):
        c = int(eg["counts"][v_i])
        if c > 1:
            P = eg["xyz"][v_i, :c].astype(np.float64)
            d = np.linalg.norm(P[:, None] - P[None, :], axis=2) + np.eye(c) * 1e9
            assert d.min() >= s * (1 - 1e-12)
    # prune + re-insert keeps working on the recycled buckets
    assert mg.prune([0, 0, 0], 12.0) == mo.prune([0, 0, 0], 12.0)
    more = _spaced_cloud(rng, 10_000)
    assert mg.insert(more) == mo.insert(more)
    _same_map(mg.export(), mo.export())
    mg.close()


def test_min_spacing_one_voxel_offered_more_points_than_the_sort_buffer():
    """20,000 offers for ONE voxel (sort buffer: 4,096): the id ranges are split; with a tiny spacing the walk goes on to the cap"""
    rng = np.random.default_rng(51)
    pts = rng.uniform(0.01, 3.99, size=(20_000, 3)).astype(np.float32)
    pts[::7] = pts[0]                                                    # exact duplicates: d2 = 0 < s2
    for s, cap in ((1e-3, 64), (1.5, 64), (0.6, 40)):
        mo, mg = oracle.Map(4.0, cap, min_spacing=s), far.Map(4.0, cap, 64, min_spacing=s)
        assert mg.insert(pts) == mo.insert(pts)
        _same_map(mg.export(), mo.export())
        mg.close()


def test_min_spacing_with_asmd_and_covariances_on_a_lidar_scan_at_the_papers_parameters():
    """v = 4 m, N_max = 40, s = v / sqrt(N_max) = 0.632 m on a ring-structured scan: contents, ids, covariance flags
    equal the oracle's; stored points really are >= 0.63 m apart; the plain insert would store clumps of consecutive ring points"""
    c2 = scenes.c2_single_frame(seed=8, n_map_candidates=60_000, map_radius=60.0, rings=32, azimuths=1024)
    v, cap, s = 4.0, 40, 4.0 / math.sqrt(40.0)
    scan, T = c2["scan"], c2["T_gt"]
    mo = oracle.Map(v, cap, min_spacing=s)
    mg = far.Map(v, cap, 1 << 14, with_cov=True, min_spacing=s)
    assert mg.insert(c2["map_points"], compute_cov=True) == mo.insert(c2["map_points"], compute_cov=True)
    assert mg.insert_asmd(scan, 30.0, 80.0, pose=T, compute_cov=True) == mo.insert_asmd(scan, 30.0, 80.0, pose=T, compute_cov=True)
    eg, eo = mg.export(with_cov=True), mo.export(with_cov=True)
    _same_map(eg, eo)
    assert np.array_equal(eg["cov_valid"], eo["cov_valid"])
    vmask = eo["cov_valid"].astype(bool)
    a, b = eg["cov"][vmask].astype(np.float64), eo["cov"][vmask].astype(np.float64)
    assert (np.linalg.norm(a - b, axis=1) / np.linalg.norm(b, axis=1)).max() < 1e-4
    dmin = np.inf
    for v_i in range(len(eg["keys"])):
        c = int(eg["counts"][v_i])
        if c > 1:
            P = eg["xyz"][v_i, :c].astype(np.float64)
            d = np.linalg.norm(P[:, None] - P[None, :], axis=2) + np.eye(c) * 1e9
            dmin = min(dmin, d.min())
    assert dmin >= 0.63
    plain = oracle.Map(v, cap)
    plain.insert(scan, pose=T)
    ep = plain.export()
    pmin = np.inf
    for v_i in range(len(ep["keys"])):
        c = int(ep["counts"][v_i])
        if c > 1:
            P = ep["xyz"][v_i, :c].astype(np.float64)
            pmin = min(pmin, (np.linalg.norm(P[:, None] - P[None, :], axis=2) + np.eye(c) * 1e9).min())
    assert pmin < 0.1                                  # consecutive ring points, centimetres apart, without the rule
    mg.close()


def test_frontend_with_regular_spacing_matches_oracle_frame():
    c2 = scenes.c2_single_frame(seed=9, n_map_candidates=80_000, map_radius=50.0, rings=16, azimuths=512)
    v, cap, s, sigma, scan = 2.0, 40, 2.0 / math.sqrt(40.0), c2["sigma"], c2["scan"]
    mo = oracle.Map(v, cap, min_spacing=s)
    mo.insert(c2["map_points"], compute_cov=True)
    ds_o, _ = oracle.voxelize(scan, 1.0)
    lo = oracle.Map(v, cap); lo.insert(scan)                              # the scan-local map of Cov-Calc is plain (R8 / R21)
    cov_o, val_o = lo.knn_cov(ds_o, nthreads=8)
    o = mo.gicp_register(ds_o, cov_o, val_o, c2["T_init"], sigma, 30, nthreads=8)
    so = mo.insert(scan, pose=(o["R"], o["t"]), compute_cov=True)
    mo.prune(o["t"], 40.0)
    fe = far.Frontend(v, cap, 1 << 15, len(scan), ds_voxel=1.0, prune_radius=40.0, max_iters=30, min_spacing=s)
    fe.map.insert(c2["map_points"], compute_cov=True)
    g = fe.process_host(scan, c2["T_init"], sigma)
    assert g["status"] == 0 and g["iters"] == o["iters"] and g["n_inliers"] == o["n_inliers"]
    assert np.linalg.norm(g["t"] - o["t"]) < 1e-4
    assert fe.insert_stats() == so
    eg, eo = fe.map.export(with_cov=True), mo.export(with_cov=True)
    assert np.array_equal(eg["keys"], eo["keys"]) and np.array_equal(eg["ids"], eo["ids"])
    assert np.abs(eg["xyz"] - eo["xyz"]).max() < 1e-5
    assert np.array_equal(eg["cov_valid"], eo["cov_valid"])
    fe.close()
