"""GPU parity at BASELINE.json's FULL sizes (configs[1..4]), in the launch configuration bench.py times.

C2: the bench step itself (far.Frontend with bench.py's parameters, one whole frame) against the oracle's frame:
    map contents after the 1.52 M-point build, downsampling, iteration/inlier counts, pose, H/b, the map after
    insert + prune -- whole outputs, not samples (the oracle finishes C2 in ~10 s).
C3: the whole 200-frame racing sequence (3 x 60k rays at 250 km/h, per-frame insert and 200 m prune) through
    far_frontend_process_host, every frame against the oracle on the same initial guess: the prior of the paper's loop
    (the EKF, driven by a synthetic IMU and corrected by the registered poses).  The literal
    constant-velocity guess of BASELINE.json is parity-tested on 14 frames at the straight-to-arc transition and on
    frames 2-41 of the bench leg's sequence (tests/test_oracle_c3.py: it is well-posed once the predicted rotation is
    kept orthonormal; the divergence reported in rounds 1-2 came from the unprojected composition).
C4: 10 M points in 100 batches of 100k, whole map compared bit for bit, then the radius prune.
C5: 20 M-point map, 1 M queries, ids and d2 bit-exact for every query at all four voxel sizes, plus brute force
    over ALL stored points on a sample (independent of the oracle's map structure).
"""
import math

import numpy as np
import pytest
import torch

import far_scenes as scenes
import oracle
from helpers import np_nn_bruteforce, rot_angle, rot_sin

pytestmark = pytest.mark.gpu

far = pytest.importorskip("paper_2606_26010_b200")


def _same_contents(g, o):
    assert np.array_equal(g["keys"], o["keys"])
    assert np.array_equal(g["counts"], o["counts"])
    assert np.array_equal(g["ids"], o["ids"])
    assert np.array_equal(g["xyz"].view(np.uint32), o["xyz"].view(np.uint32))


def _cov_close(g, o, tol=1e-4):
    assert np.array_equal(g["cov_valid"], o["cov_valid"])
    v = o["cov_valid"].astype(bool)
    a, b = g["cov"][v].astype(np.float64), o["cov"][v].astype(np.float64)
    rel = np.linalg.norm(a - b, axis=1) / np.linalg.norm(b, axis=1)
    assert rel.max() < tol, rel.max()


# Stored coordinates after an insert at a REGISTERED pose.  A stored coordinate is the pose applied to the point in FP64,
# rounded to fp32 once.  The two sides' poses agree to ~1e-10 ... 1e-8 m (different summation orders of the same FP64 terms,
# amplified by the chain of frames), which moves the FP64 value by at most  |dt| + sin(angle) x range  -- the POSE SLACK, taken
# from the very poses the test compares, frame by frame -- and the rounding then adds at most one fp32 ulp of the value
# (neighbouring fp32 numbers where the slack straddles a rounding boundary).  So the bar is one ulp of the value plus the
# measured pose slack, not a number of metres picked for the scene.  (At a GIVEN pose the same insert is bit-exact:
# tests/test_gpu_map.py.)
MAX_RANGE_M = 200.0


def _pose_slack(g, o):
    return float(np.linalg.norm(g["t"] - o["t"])) + rot_sin(g["R"].T @ o["R"]) * MAX_RANGE_M


def _xyz_within_one_ulp_plus(g, o, slack):
    assert slack < 1e-6, slack                                   # the poses themselves are far inside north_star's 1e-4 m
    g, o = np.ascontiguousarray(g), np.ascontiguousarray(o)
    d = np.abs(g.astype(np.float64) - o.astype(np.float64))
    ulp = np.spacing(np.maximum(np.abs(g), np.abs(o))).astype(np.float64)
    worst = (d - ulp).max()
    assert worst <= slack, (float(worst), slack, float((d > 0).mean()))


def _result(d_res):
    return far.result_to_dict(far.GicpResult.from_buffer_copy(d_res.cpu().numpy().tobytes()))


def test_c2_full_frame_as_benched():
    import bench
    c2 = bench.load_workload("c2")
    scan, v, cap, sigma = c2["scan"], c2["voxel"], c2["cap"], c2["sigma"]
    # ---- oracle frame ----
    mo = oracle.Map(v, cap)
    so = mo.insert(c2["map_points"], compute_cov=True)
    eo0 = mo.export(with_cov=True)
    ds_o, idx_o = oracle.voxelize(scan, v)
    lo = oracle.Map(v, cap)
    lo.insert(scan)
    cov_o, val_o = lo.knn_cov(ds_o, nthreads=16)
    o = mo.gicp_register(ds_o, cov_o, val_o, c2["T_init"], sigma, bench.MAX_ITERS, nthreads=16)
    # ---- CUDA path: exactly bench.py's construction and step ----
    fe = far.Frontend(v, cap, c2["max_voxels"], len(scan), ds_voxel=v, prune_radius=bench.PRUNE_RADIUS,
                      max_iters=bench.MAX_ITERS)
    sg = fe.map.insert(torch.as_tensor(c2["map_points"]).cuda(), compute_cov=True)
    assert sg == so
    eg0 = fe.map.export(with_cov=True)
    _same_contents(eg0, eo0)
    _cov_close(eg0, eo0)
    # NN on the full map: every downsampled scan point at the true pose, bit-exact; brute force on a sample
    q = scenes.pose_apply(c2["T_gt"], ds_o)
    ids_o, d2_o = mo.nn(q)
    ids_g, d2_g = fe.map.nn(q)
    assert np.array_equal(ids_g.cpu().numpy().view(np.uint32), ids_o)
    assert np.array_equal(d2_g.cpu().numpy().view(np.uint32), d2_o.view(np.uint32))
    stored = eo0["counts"][:, None] > np.arange(cap)[None, :]
    sel = np.random.default_rng(0).choice(len(q), 64, replace=False)
    bf_ids, _ = np_nn_bruteforce(eo0["xyz"][stored], eo0["ids"][stored], q[sel], v)
    assert np.array_equal(ids_g.cpu().numpy().view(np.uint32)[sel], bf_ids)
    # one linearisation at the initial pose: H, b
    vox_xyz, vox_idx = far.voxelize(torch.as_tensor(scan).cuda(), v)
    assert np.array_equal(vox_idx.cpu().numpy(), idx_o)
    lg = far.Map(v, cap, len(scan))
    lg.insert(scan)
    cov_g, val_g = lg.knn_cov(vox_xyz)
    assert np.array_equal(val_g.cpu().numpy(), val_o)
    lin_o = mo.gicp_linearize(ds_o, cov_o, val_o, c2["T_init"], sigma)
    lin_g = fe.map.gicp_linearize(vox_xyz, cov_g, val_g, c2["T_init"], sigma)
    assert lin_g["n_inliers"] == lin_o["n_inliers"]
    assert np.linalg.norm(lin_g["H"] - lin_o["H"]) / np.linalg.norm(lin_o["H"]) < 1e-4
    assert np.linalg.norm(lin_g["b"] - lin_o["b"]) / np.linalg.norm(lin_o["b"]) < 1e-4
    # the benched step
    d_res = torch.zeros(far.GICP_RESULT_BYTES, dtype=torch.uint8, device="cuda")
    fe.process_enqueue(torch.as_tensor(scan).cuda(), c2["T_init"], sigma, d_result=d_res)
    torch.cuda.synchronize()
    g = _result(d_res)
    assert g["status"] == o["status"] == 0
    assert g["iters"] == o["iters"] and g["n_inliers"] == o["n_inliers"] and g["converged"] == o["converged"]
    assert np.linalg.norm(g["t"] - o["t"]) < 1e-4 and rot_angle(g["R"].T @ o["R"]) < 1e-5
    assert np.linalg.norm(g["H"] - o["H"]) / np.linalg.norm(o["H"]) < 1e-4
    # map update at the registered pose + prune
    mo.insert(scan, pose=(o["R"], o["t"]), compute_cov=True)
    mo.prune(o["t"], bench.PRUNE_RADIUS)
    eo1, eg1 = mo.export(with_cov=True), fe.map.export(with_cov=True)
    assert np.array_equal(eg1["keys"], eo1["keys"]) and np.array_equal(eg1["counts"], eo1["counts"])
    assert np.array_equal(eg1["ids"], eo1["ids"])
    _xyz_within_one_ulp_plus(eg1["xyz"], eo1["xyz"], _pose_slack(g, o))
    assert np.array_equal(eg1["cov_valid"], eo1["cov_valid"])
    fe.close()


@pytest.mark.parametrize("s0,n_frames", [(990.0, 14), (300.0, 42)])
def test_c3_racing_frames_chain_matches_oracle_frame_by_frame(s0, n_frames):
    """The literal constant-velocity guess of BASELINE.json configs[2], T_pred = T_{t-1} (T_{t-2}^-1 T_{t-1}) with the rotation
    projected back onto SO(3) (tests/test_oracle_c3.py shows why: without the projection the composition loses orthonormality
    geometrically and the sequence diverges after ~30 frames -- the "drift" rounds 1-2 attributed to the method).
    s0 = 990: the end of the straight and the entry of the R = 500 m arc, iteration counts from 2 to 30.
    s0 = 300: the start of the bench leg's sequence, frames 2-41.
    Same status, iterations, inliers and pose on every frame, same map at the end."""
    v, cap, prune_r, max_range = 1.0, 20, 200.0, 200.0
    track = scenes.RaceTrack(seed=2)
    rng = np.random.default_rng(2)
    step = 69.4 * 0.1                      # 250 km/h at 10 Hz
    frames = [scenes.c3_racing_frame(track, s0 + step * f, rng) for f in range(n_frames)]
    n_max = max(len(s) for s, _ in frames)
    fe = far.Frontend(v, cap, 1 << 19, n_max, ds_voxel=v, prune_radius=prune_r, max_iters=30)
    mo = oracle.Map(v, cap)
    th_o, th_g = oracle.AdaptiveThreshold(2.0, 0.1, max_range), far.AdaptiveThreshold(2.0, 0.1, max_range)
    # bootstrap: two frames inserted at their ground-truth poses (gives the constant-velocity model its velocity)
    poses_o, poses_g = [], []
    for f in range(2):
        scan, T = frames[f]
        assert fe.map.insert(scan, pose=T, compute_cov=True) == mo.insert(scan, pose=T, compute_cov=True)
        poses_o.append(T)
        poses_g.append(T)

    def predict(P):   # T_pred = T_{t-1} (T_{t-2}^-1 T_{t-1}), projected back onto SO(3): the product of three matrices with a
        # transpose for the inverse multiplies any deviation from orthonormality from frame to frame (1e-11 in the
        # bootstrap poses had grown to 2e-8 by frame 22 of the long run), and a predicted pose is a rigid transform
        R, t = scenes.pose_compose(P[-1], scenes.pose_compose(scenes.pose_inverse(P[-2]), P[-1]))
        U, _, Vt = np.linalg.svd(R)
        return U @ Vt, t

    iters, slack = [], 0.0
    for f in range(2, n_frames):
        scan, T_gt = frames[f]
        pred_o, pred_g = predict(poses_o), predict(poses_g)
        ds_o, _ = oracle.voxelize(scan, v)
        lo = oracle.Map(v, cap)
        lo.insert(scan)
        cov_o, val_o = lo.knn_cov(ds_o, nthreads=16)
        o = mo.gicp_register(ds_o, cov_o, val_o, pred_o, th_o.sigma(), 30, nthreads=16)
        mo.insert(scan, pose=(o["R"], o["t"]), compute_cov=True)
        mo.prune(o["t"], prune_r)
        g = fe.process_host(scan, pred_g, th_g.sigma())
        assert g["status"] == o["status"] == 0, f
        assert g["n_inliers"] == o["n_inliers"] and g["iters"] == o["iters"] and g["converged"] == o["converged"], f
        # sin of the angle from the antisymmetric part (helpers.rot_sin): well-conditioned at 1e-5 rad and below
        assert np.linalg.norm(g["t"] - o["t"]) < 1e-4 and rot_sin(g["R"].T @ o["R"]) < 1e-5, f
        for R in (g["R"], o["R"]):
            assert np.abs(R.T @ R - np.eye(3)).max() < 1e-9, f
        slack = max(slack, _pose_slack(g, o))
        th_o.update(pred_o, (o["R"], o["t"]))
        th_g.update(pred_g, (g["R"], g["t"]))
        assert abs(th_o.sigma() - th_g.sigma()) < 1e-6
        poses_o.append((o["R"], o["t"]))
        poses_g.append((g["R"], g["t"]))
        assert mo.size() == fe.map.size(), f
        iters.append(o["iters"])
    assert min(iters) < 10 and max(iters) > (10 if s0 == 990.0 else 7)     # both quick and long registrations were exercised
    eo, eg = mo.export(with_cov=True), fe.map.export(with_cov=True)
    assert np.array_equal(eg["keys"], eo["keys"]) and np.array_equal(eg["ids"], eo["ids"])
    _xyz_within_one_ulp_plus(eg["xyz"], eo["xyz"], slack)
    assert np.array_equal(eg["cov_valid"], eo["cov_valid"])
    # the corridor is degenerate along-track (expect it, report it, do not tune it away):
    # only lateral / vertical / heading errors are bounded
    R, t = poses_g[-1]
    Rg, tg = frames[-1][1]
    err = Rg.T @ (t - tg)
    assert rot_angle(R.T @ Rg) < math.radians(0.5)
    if s0 == 990.0:
        assert np.abs(err[1:]).max() < 0.1
    else:   # well-posed on the straight, as on the oracle (test_oracle_c3.py); height is held by the road surface only and
        # wanders by a few decimetres over 40 frames on both sides alike
        assert abs(err[0]) < 0.2 and abs(err[1]) < 0.1 and abs(err[2]) < 0.5 and th_g.sigma() < 0.3
    fe.close()


def test_c3_racing_sequence_200_frames_ekf_prior_matches_oracle_every_frame():
    """BASELINE.json configs[2] at its configured length.  One loop produces the initial guesses (the product's: far_ekf_*
    fed with the GPU's registered poses and Eq. 7 velocities, 20 ms late, up-sampled over 5 cycles); the oracle registers
    every frame from the same guess and the same sigma against ITS OWN map.  Asserted per frame: status, iteration count,
    inlier count, pose; at the end: the whole map.  Reported: drift of both sides against ground truth."""
    n_frames, v, cap, prune_r, vel, dt, s0 = 200, 1.0, 20, 200.0, 69.4, 0.01, 300.0
    G0 = 9.80665
    track = scenes.RaceTrack(seed=2)
    rng = np.random.default_rng(2)
    frames = [scenes.c3_racing_frame(track, s0 + 6.94 * f, rng) for f in range(n_frames)]
    n_max = max(len(s) for s, _ in frames)
    fe = far.Frontend(v, cap, 1 << 16, n_max, ds_voxel=v, prune_radius=prune_r, max_iters=30)
    mo = oracle.Map(v, cap)
    th_g, th_o = far.AdaptiveThreshold(2.0, 0.1, 200.0), oracle.AdaptiveThreshold(2.0, 0.1, 200.0)
    for f in range(2):
        assert fe.map.insert(frames[f][0], pose=frames[f][1], compute_cov=True) == mo.insert(frames[f][0], pose=frames[f][1], compute_cov=True)

    def yaw_rate(cycle):
        return vel / track.radius if s0 + vel * dt * cycle > track.straight else 0.0

    T1 = frames[1][1]
    ekf = far.Ekf(np.r_[T1[1], 0.0, 0.0, 0.0, vel, 0.0, 0.0], [0.05] * 3 + [1e-4] * 3 + [0.1] * 3,
                  [1e-6] * 3 + [1e-8] * 3 + [1e-4] * 3, dt=dt, n_up=5)
    Rz = [4e-4] * 3 + [1e-6] * 3 + [0.25] * 3
    irng = np.random.default_rng(7)
    cycle, T_prev = 10, T1

    def imu_step():
        nonlocal cycle
        w = yaw_rate(cycle)
        ekf.predict(np.r_[0.0, vel * w, G0] + irng.normal(0, 0.05, 3), np.r_[0.0, 0.0, w] + irng.normal(0, 0.002, 3))
        cycle += 1

    iters, err_g, err_o, dmax, slack = [], [], [], 0.0, 0.0
    for f in range(2, n_frames):
        scan, T_gt = frames[f]
        while cycle < 10 * f:
            imu_step()
        pred, sigma = ekf.pose(), th_g.sigma()
        g = fe.process_host(scan, pred, sigma)
        ds_o, _ = oracle.voxelize(scan, v)
        lo = oracle.Map(v, cap)
        lo.insert(scan)
        cov_o, val_o = lo.knn_cov(ds_o, nthreads=16)
        o = mo.gicp_register(ds_o, cov_o, val_o, pred, sigma, 30, nthreads=16)
        mo.insert(scan, pose=(o["R"], o["t"]), compute_cov=True)
        mo.prune(o["t"], prune_r)
        assert g["status"] == o["status"] == 0, f
        assert g["n_inliers"] == o["n_inliers"] and g["iters"] == o["iters"] and g["converged"] == o["converged"], f
        assert np.linalg.norm(g["t"] - o["t"]) < 1e-4 and rot_angle(g["R"].T @ o["R"]) < 1e-5, f
        dmax = max(dmax, float(np.linalg.norm(g["t"] - o["t"])))
        slack = max(slack, _pose_slack(g, o))
        th_g.update(pred, (g["R"], g["t"])); th_o.update(pred, (o["R"], o["t"]))
        assert abs(th_g.sigma() - th_o.sigma()) < 1e-6
        assert mo.size() == fe.map.size(), f
        T_L = (g["R"], g["t"])
        v_L = far.lidar_velocity(T_L, T_prev, 0.1)              # Eq. 7
        T_prev = T_L
        imu_step(); imu_step()                                   # the result reaches the EKF 20 ms later
        ekf.push_lidar(T_L, v_L, Rz, cycle_s=10 * f - 10)
        err_g.append(T_gt[0].T @ (g["t"] - T_gt[1])); err_o.append(T_gt[0].T @ (o["t"] - T_gt[1]))
        iters.append(o["iters"])
    eo, eg = mo.export(with_cov=True), fe.map.export(with_cov=True)
    assert np.array_equal(eg["keys"], eo["keys"]) and np.array_equal(eg["counts"], eo["counts"])
    assert np.array_equal(eg["ids"], eo["ids"])
    _xyz_within_one_ulp_plus(eg["xyz"], eo["xyz"], slack)
    assert np.array_equal(eg["cov_valid"], eo["cov_valid"])
    st = fe.map.stats()
    assert st["full"] == 0 and st["n_rehash"] > 0 and st["n_dead_keys"] < 64 + st["n_voxels"] // 4    # 2^16-bucket map, 198 prunes
    drift_g, drift_o = np.abs(np.array(err_g)).max(axis=0), np.abs(np.array(err_o)).max(axis=0)
    print(f"C3 200 frames: max |t_gpu - t_oracle| = {dmax:.2e} m; iterations {min(iters)}..{max(iters)}; "
          f"max drift along/lateral/vertical GPU {drift_g.round(3)} oracle {drift_o.round(3)} m")
    assert np.allclose(drift_g, drift_o, atol=1e-3)
    assert drift_g[1] < 0.5 and max(iters) < 30           # stays on the track, never hits the iteration limit
    fe.close()


def test_c4_insert_stress_full_10m_points_in_100_batches_then_prune():
    pts = scenes.c4_insert_stress(seed=3)
    assert pts.shape == (10_000_000, 3)
    v, cap = 0.5, 20
    mo = oracle.Map(v, cap)
    so = mo.insert(pts)                                         # batch invariance of the oracle is pinned on CPU
    mg = far.Map(v, cap, 9_000_000, with_cov=False, max_batch=100_000)
    d_pts = torch.as_tensor(pts).cuda()
    acc = dict(n_offered=0, n_accepted=0, n_new_voxels=0, n_dropped_full=0, n_invalid=0)
    for b in range(100):
        st = mg.insert(d_pts[b * 100_000:(b + 1) * 100_000])
        for k in acc:
            acc[k] += st[k]
    assert acc == so
    assert mg.size() == mo.size()
    _same_contents(mg.export(), mo.export())
    po = mo.prune([0.0, 0.0, 0.0], 150.0)
    pg = mg.prune([0.0, 0.0, 0.0], 150.0)
    assert pg == po and po["n_voxels_removed"] > 0
    eg, eo = mg.export(), mo.export()
    assert np.array_equal(eg["keys"], eo["keys"]) and np.array_equal(eg["ids"], eo["ids"])
    mg.close()


@pytest.fixture(scope="module")
def c5_workload():
    return scenes.c5_nn_sweep(seed=4)


@pytest.mark.parametrize("voxel", [1.0, 0.25, 0.5, 2.0])
def test_c5_nn_sweep_full_20m_map_1m_queries(voxel, c5_workload):
    c5 = c5_workload
    pts, q = c5["map_points"], c5["queries"]
    assert len(pts) == 20_000_000 and len(q) == 1_000_000
    cap = 20
    mo = oracle.Map(voxel, cap)
    so = mo.insert(pts)
    mg = far.Map(voxel, cap, so["n_new_voxels"] + 1024, with_cov=False, max_batch=1 << 22)
    sg = mg.insert(torch.as_tensor(pts).cuda())
    assert sg == so
    ids_o, d2_o = mo.nn(q, nthreads=16)
    for order in (c5["order"], c5["morton_order"]):
        qq = np.ascontiguousarray(q[order])
        ids_g, d2_g = mg.nn(torch.as_tensor(qq).cuda())
        assert np.array_equal(ids_g.cpu().numpy().view(np.uint32), ids_o[order])
        assert np.array_equal(d2_g.cpu().numpy().view(np.uint32), d2_o[order].view(np.uint32))
    hit = ids_o != 0xFFFFFFFF
    assert 0.45 < hit.mean() < 1.0 and (~hit[~c5["is_hit"]]).any()
    # brute force over ALL offered points (stored ones = first `cap` per voxel are what NN may return: use ids)
    e = mo.export()
    stored = e["counts"][:, None] > np.arange(cap)[None, :]
    sel = np.random.default_rng(1).choice(len(q), 24, replace=False)
    bf_ids, bf_d2 = np_nn_bruteforce(e["xyz"][stored], e["ids"][stored], q[sel], voxel)
    ids_g, d2_g = mg.nn(torch.as_tensor(np.ascontiguousarray(q[sel])).cuda())
    assert np.array_equal(ids_g.cpu().numpy().view(np.uint32), bf_ids)
    assert np.array_equal(d2_g.cpu().numpy(), bf_d2.astype(np.float32))
    mg.close()
