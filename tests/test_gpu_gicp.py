"""GPU parity: k-NN covariances (Eq. 1), one GICP linearisation (H, b) and the registration loop -- CUDA path
through the C ABI vs the FP64 CPU oracle.  Tolerances are BASELINE.json's north_star: covariance valid flags
bit-exact, Sigma and H/b within 1e-4 relative, converged poses within 1e-4 m / 1e-5 rad."""
import math

import numpy as np
import pytest
import torch

import far_scenes as scenes
import oracle
from helpers import load_golden, rot_angle

pytestmark = pytest.mark.gpu

far = pytest.importorskip("paper_2606_26010_b200")

KERNELS = [oracle.KERNEL_CAUCHY, oracle.KERNEL_GEMAN_MCCLURE, oracle.KERNEL_NONE]


def _rel_cov(a, b):
    a, b = a.astype(np.float64), b.astype(np.float64)
    return np.linalg.norm(a - b, axis=-1) / np.linalg.norm(b, axis=-1)


def _hb_err(g, o, scale_b):
    eh = np.linalg.norm(g["H"] - o["H"]) / np.linalg.norm(o["H"])
    eb = np.linalg.norm(g["b"] - o["b"]) / max(np.linalg.norm(o["b"]), 1e-3 * scale_b)
    return eh, eb


def _pose_err(g, o):
    dt = np.linalg.norm(g["t"] - o["t"])
    dr = rot_angle(g["R"].T @ o["R"])
    return dt, dr


def _build_pair(map_points, voxel, cap, max_voxels=None):
    mo = oracle.Map(voxel, cap)
    mg = far.Map(voxel, cap, max_voxels or 4 * len(map_points) + 1024, with_cov=True)
    so = mo.insert(map_points, compute_cov=True)
    sg = mg.insert(map_points, compute_cov=True)
    assert sg == so
    return mo, mg


def _scan_cov(scan_raw, scan_ds, voxel, cap):
    """Sigma_s from a scan-local map built from the raw scan, on both sides."""
    lo = oracle.Map(voxel, cap)
    lo.insert(scan_raw)
    cov_o, val_o = lo.knn_cov(scan_ds, nthreads=8)
    lg = far.Map(voxel, cap, 4 * len(scan_raw) + 1024)
    lg.insert(scan_raw)
    cov_g, val_g = lg.knn_cov(scan_ds)
    return (cov_o, val_o), (cov_g, val_g)


# ---- A7 ---------------------------------------------------------------------------------------------------
def test_cov_closed_form_golden():
    g = load_golden("cov_eq1_closed_form.json")
    # eight points (the corners (+-a, +-a, 0), twice) whose 1/k sample covariance is diag(0.1, 0.1, 0)
    a = math.sqrt(0.1)
    corners = np.array([[a, a, 0], [a, -a, 0], [-a, a, 0], [-a, -a, 0]], dtype=np.float64)
    pts = (np.concatenate([corners, corners]) + 1.0).astype(np.float32)      # all inside voxel (0,0,0) of a 4 m grid
    mg = far.Map(4.0, 20, 64, k_cov=8, cov_eps=g["eps"])
    mg.insert(pts)
    cov, valid = mg.knn_cov(pts[:1])
    assert int(valid[0]) == 1
    c = cov[0].cpu().numpy().astype(np.float64)
    S = np.array([[c[0], c[1], c[2]], [c[1], c[3], c[4]], [c[2], c[4], c[5]]])
    assert np.allclose(np.sort(np.linalg.eigvalsh(S)), np.sort(g["eig_sigma"]), rtol=1e-5)
    assert np.linalg.norm(np.linalg.inv(S)) == pytest.approx(1.0, rel=1e-5)        # ||Sigma^-1||_F = 1 (Eq. 1)
    # fewer than k neighbours -> invalid, identity
    mg2 = far.Map(4.0, 20, 64, k_cov=10)
    mg2.insert(pts)
    cov, valid = mg2.knn_cov(pts[:1])
    assert int(valid[0]) == 0 and cov[0].tolist() == [1, 0, 0, 1, 0, 1]


@pytest.mark.parametrize("voxel,cap,k", [(0.5, 20, 10), (1.0, 20, 10), (1.0, 40, 10), (0.5, 4, 5)])
def test_knn_cov_matches_oracle(voxel, cap, k):
    c1 = scenes.c1_tiny(seed=3, n_map=20_000, n_scan=3001)
    mo = oracle.Map(voxel, cap, k_cov=k)
    mg = far.Map(voxel, cap, 100_000, k_cov=k)
    mo.insert(c1["map_points"]); mg.insert(c1["map_points"])
    rng = np.random.default_rng(1)
    q = np.concatenate([c1["map_points"][:2000], scenes.pose_apply(c1["T_gt"], c1["scan"]),
                        rng.uniform(-8, 8, (500, 3)).astype(np.float32)]).astype(np.float32)
    cov_o, val_o = mo.knn_cov(q, nthreads=8)
    cov_g, val_g = mg.knn_cov(q)
    assert np.array_equal(val_g.cpu().numpy(), val_o)
    assert val_o.any() and not val_o.all()
    v = val_o.astype(bool)
    assert _rel_cov(cov_g.cpu().numpy()[v], cov_o[v]).max() < 1e-4
    assert np.array_equal(cov_g.cpu().numpy()[~v], cov_o[~v])              # identity where invalid


def test_insert_compute_cov_matches_oracle_across_batches():
    c1 = scenes.c1_tiny(seed=4, n_map=30_000)
    pts = c1["map_points"]
    mo, mg = oracle.Map(0.5, 20), far.Map(0.5, 20, 100_000, with_cov=True)
    for a, b in [(0, 10_000), (10_000, 10_001), (10_001, 30_000)]:      # covariances are NOT batch invariant: replay
        so = mo.insert(pts[a:b], compute_cov=True)
        sg = mg.insert(pts[a:b], compute_cov=True)
        assert sg == so
    eo, eg = mo.export(with_cov=True), mg.export(with_cov=True)
    assert np.array_equal(eg["keys"], eo["keys"]) and np.array_equal(eg["ids"], eo["ids"])
    assert np.array_equal(eg["cov_valid"], eo["cov_valid"])
    v = eo["cov_valid"].astype(bool)
    assert v.any()
    assert _rel_cov(eg["cov"][v], eo["cov"][v]).max() < 1e-4
    # the oversize path (call larger than the covariance queue) gives the same covariances
    mc = far.Map(0.5, 20, 100_000, with_cov=True, max_batch=4096)
    for a, b in [(0, 10_000), (10_000, 10_001), (10_001, 30_000)]:
        mc.insert(pts[a:b], compute_cov=True)
    ec = mc.export(with_cov=True)
    assert np.array_equal(ec["cov_valid"], eo["cov_valid"])
    assert _rel_cov(ec["cov"][v], eo["cov"][v]).max() < 1e-4


@pytest.mark.parametrize("voxel,cap,k", [(0.5, 20, 12), (1.0, 64, 10), (2.0, 64, 16), (0.5, 8, 3), (1.0, 33, 10)])
def test_insert_compute_cov_task_kernel_paths(voxel, cap, k):
    """The one-warp-per-touched-voxel covariance kernel off its main road: k > 10 (every query takes the warp-level exact
    selection), cap 64 with voxels that receive more than 32 points in one call (two passes of queries, one lane per query),
    small k, a cap that is not a multiple of 4 -- in two batches, both through the task list and through the oversize path."""
    c1 = scenes.c1_tiny(seed=6, n_map=40_000)
    pts = c1["map_points"]
    mo = oracle.Map(voxel, cap, k_cov=k)
    mg = far.Map(voxel, cap, 100_000, with_cov=True, k_cov=k)
    mc = far.Map(voxel, cap, 100_000, with_cov=True, k_cov=k, max_batch=4096)      # oversize path: knn_cov_new_ids_kernel
    for a, b in [(0, 25_000), (25_000, 40_000)]:
        assert mg.insert(pts[a:b], compute_cov=True) == mo.insert(pts[a:b], compute_cov=True)
        mc.insert(pts[a:b], compute_cov=True)
    eo, eg, ec = mo.export(with_cov=True), mg.export(with_cov=True), mc.export(with_cov=True)
    assert np.array_equal(eg["keys"], eo["keys"]) and np.array_equal(eg["ids"], eo["ids"])
    assert np.array_equal(eg["cov_valid"], eo["cov_valid"]) and np.array_equal(ec["cov_valid"], eo["cov_valid"])
    v = eo["cov_valid"].astype(bool)
    assert v.any()
    if cap == 64:
        assert eo["counts"].max() > 32                                   # a voxel did receive more than a warp's worth
    assert _rel_cov(eg["cov"][v], eo["cov"][v]).max() < 1e-4
    assert _rel_cov(ec["cov"][v], eo["cov"][v]).max() < 1e-4


def test_insert_compute_cov_on_a_lattice_with_distance_ties():
    """Lattice points: every query has exact distance ties across its 10th..12th neighbours, so the coarse-key proof fails
    everywhere and the exact selection (ties broken by the lowest id, R6) decides -- valid flags and covariances as the oracle's."""
    g = np.arange(-6, 6, dtype=np.float32) * np.float32(0.25)
    pts = np.stack(np.meshgrid(g, g, g[:6], indexing="ij"), axis=-1).reshape(-1, 3).astype(np.float32)
    rng = np.random.default_rng(0)
    pts = pts[rng.permutation(len(pts))]
    mo, mg = oracle.Map(1.0, 20), far.Map(1.0, 20, 4096, with_cov=True)
    assert mg.insert(pts, compute_cov=True) == mo.insert(pts, compute_cov=True)
    eo, eg = mo.export(with_cov=True), mg.export(with_cov=True)
    assert np.array_equal(eg["ids"], eo["ids"]) and np.array_equal(eg["cov_valid"], eo["cov_valid"])
    v = eo["cov_valid"].astype(bool)
    assert v.any()
    assert _rel_cov(eg["cov"][v], eo["cov"][v]).max() < 1e-4


# ---- A8-A10 ----------------------------------------------------------------------------------------------
def test_single_correspondence_and_robust_weight_golden():
    g = load_golden("gicp_single_correspondence.json")
    mg = far.Map(0.5, 20, 64, with_cov=True)
    mg.insert(np.array([g["r"]], dtype=np.float32))
    scan = np.array([g["p"]], dtype=np.float32)
    res = mg.gicp_linearize(scan, None, None, scenes.pose_identity(), 2.0, far.default_options(kernel=far.KERNEL_NONE))
    assert res["n_inliers"] == 1 and res["iters"] == 1
    assert np.allclose(res["H"], np.array(g["H"], dtype=np.float64), atol=1e-7)
    assert np.allclose(res["b"], np.array(g["b"]), atol=1e-7)
    # robust weights (Eq. 5 and the kernel of [1]): M = I, e2 = |d|^2 = 0.01, sigma = 1 -> kappa = 1/3; H[0,0] = w
    w = load_golden("robust_weights.json")
    for kernel, name in [(far.KERNEL_CAUCHY, "cauchy"), (far.KERNEL_GEMAN_MCCLURE, "geman_mcclure"), (far.KERNEL_NONE, "none")]:
        res = mg.gicp_linearize(scan, None, None, scenes.pose_identity(), 1.0, far.default_options(kernel=kernel))
        e2 = float(np.float32(0.1)) ** 2
        want = {"cauchy": 1 / (1 + e2 * 9), "geman_mcclure": (1 / 9) / (1 / 3 + e2) ** 2, "none": 1.0}[name]
        assert res["H"][0, 0] == pytest.approx(want, rel=1e-12)
        assert res["H"][0, 0] == pytest.approx(w[name], rel=1e-6)
    # gate: tau = 3 sigma; sigma = 0.03 -> tau = 0.09 < 0.1 rejects the only correspondence
    res = mg.gicp_linearize(scan, None, None, scenes.pose_identity(), 0.03)
    assert res["n_inliers"] == 0 and np.all(res["H"] == 0)


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("sigma", [2.0, 0.05])
def test_linearize_matches_oracle_c1(kernel, sigma):
    c1 = scenes.c1_tiny(seed=0)
    mo, mg = _build_pair(c1["map_points"], c1["voxel"], c1["cap"])
    (cov_o, val_o), (cov_g, val_g) = _scan_cov(c1["scan"], c1["scan"], c1["voxel"], c1["cap"])
    assert np.array_equal(val_g.cpu().numpy(), val_o)
    opts_o, opts_g = oracle.default_options(kernel=kernel), far.default_options(kernel=kernel)
    rng = np.random.default_rng(2)
    poses = [c1["T_init"], c1["T_gt"], scenes.perturb_pose(c1["T_gt"], 0.05, 0.3, rng)]
    for ip, T in enumerate(poses):
        o = mo.gicp_linearize(c1["scan"], cov_o, val_o, T, sigma, opts_o)
        g = mg.gicp_linearize(c1["scan"], cov_g, val_g, T, sigma, opts_g)
        assert g["n_inliers"] == o["n_inliers"] and o["n_inliers"] > 0
        corr = mo.gicp_correspondences(c1["scan"], cov_o, val_o, T, sigma, opts_o)
        # scale for b: sum of the per-correspondence gradient norms (b itself -> 0 at convergence)
        d = corr["r"] - corr["p"]
        Md = np.einsum("nij,nj->ni", corr["M"], d)
        scale_b = float(np.sum(corr["w"][corr["used"]] * np.linalg.norm(Md[corr["used"]], axis=1)))
        eh, eb = _hb_err(g, o, scale_b)
        assert eh < 1e-4 and eb < 1e-4, (eh, eb)
        assert g["chi2"] == pytest.approx(o["chi2"], rel=1e-6)
        if sigma < 1.0 and ip == 0:
            assert o["n_inliers"] < len(c1["scan"])          # the gate (tau = 0.15 m) rejects something at T_init


@pytest.mark.parametrize("kernel", KERNELS)
def test_register_matches_oracle_c1(kernel):
    c1 = scenes.c1_tiny(seed=0)
    mo, mg = _build_pair(c1["map_points"], c1["voxel"], c1["cap"])
    (cov_o, val_o), (cov_g, val_g) = _scan_cov(c1["scan"], c1["scan"], c1["voxel"], c1["cap"])
    # fixed point (eps = 1e-6): both sides sit at the same minimum
    oo, og = oracle.default_options(kernel=kernel, conv_eps=1e-6), far.default_options(kernel=kernel, conv_eps=1e-6)
    o = mo.gicp_register(c1["scan"], cov_o, val_o, c1["T_init"], c1["sigma"], c1["max_iters"], oo, nthreads=8)
    g = mg.gicp_register(c1["scan"], cov_g, val_g, c1["T_init"], c1["sigma"], c1["max_iters"], og)
    assert g["status"] == o["status"] == 0
    dt, dr = _pose_err(g, o)
    assert dt < 1e-4 and dr < 1e-5, (dt, dr)
    assert g["converged"] == o["converged"] and abs(g["iters"] - o["iters"]) <= 1
    # the paper's eps = 5e-3: same iteration count, same pose
    oo, og = oracle.default_options(kernel=kernel), far.default_options(kernel=kernel)
    o = mo.gicp_register(c1["scan"], cov_o, val_o, c1["T_init"], c1["sigma"], c1["max_iters"], oo, nthreads=8)
    g = mg.gicp_register(c1["scan"], cov_g, val_g, c1["T_init"], c1["sigma"], c1["max_iters"], og)
    assert g["iters"] == o["iters"] and g["converged"] == o["converged"] == 1
    dt, dr = _pose_err(g, o)
    assert dt < 1e-4 and dr < 1e-5
    assert g["n_inliers"] == o["n_inliers"]
    eh, eb = _hb_err(g, o, np.linalg.norm(o["H"]))
    assert eh < 1e-4
    # and it found the ground truth to scan-noise level
    dt, dr = _pose_err(g, dict(R=c1["T_gt"][0], t=c1["T_gt"][1]))
    assert dt < 0.01 and dr < math.radians(0.1)


@pytest.mark.parametrize("n_scan", [5921, 12_000, 40_003])
def test_register_more_source_points_than_the_grid_holds_at_once(n_scan):
    """gicp_kernel keeps one source point per 16-lane group while the scan fits the grid (148 blocks x 40 points on a
    B200); beyond that it serves the points in rounds and fetches them again every iteration.  Linearisation and the whole
    registration against the oracle on scans of one point past that limit, two rounds and seven rounds, stride 3 and 4."""
    c1 = scenes.c1_tiny(seed=7, n_map=30_000, n_scan=n_scan)
    mo, mg = _build_pair(c1["map_points"], c1["voxel"], c1["cap"])
    (cov_o, val_o), (cov_g, val_g) = _scan_cov(c1["scan"], c1["scan"], c1["voxel"], c1["cap"])
    lo = mo.gicp_linearize(c1["scan"], cov_o, val_o, c1["T_init"], c1["sigma"], oracle.default_options())
    lg = mg.gicp_linearize(c1["scan"], cov_g, val_g, c1["T_init"], c1["sigma"], far.default_options())
    assert lg["n_inliers"] == lo["n_inliers"] > n_scan // 2
    eh, eb = _hb_err(lg, lo, np.linalg.norm(lo["H"]))
    assert eh < 1e-4 and eb < 1e-4
    o = mo.gicp_register(c1["scan"], cov_o, val_o, c1["T_init"], c1["sigma"], c1["max_iters"], oracle.default_options(), nthreads=16)
    g = mg.gicp_register(c1["scan"], cov_g, val_g, c1["T_init"], c1["sigma"], c1["max_iters"], far.default_options())
    assert g["status"] == o["status"] == 0 and g["iters"] == o["iters"] and g["converged"] == o["converged"] == 1
    assert g["n_inliers"] == o["n_inliers"]
    dt, dr = _pose_err(g, o)
    assert dt < 1e-4 and dr < 1e-5
    scan4 = np.concatenate([c1["scan"], np.full((n_scan, 1), 7.0, np.float32)], axis=1)
    g4 = mg.gicp_register(scan4, cov_g, val_g, c1["T_init"], c1["sigma"], c1["max_iters"], far.default_options())
    assert g4["iters"] == g["iters"] and np.array_equal(g4["t"], g["t"]) and np.array_equal(g4["H"], g["H"])


def test_noise_free_recovery_and_point_to_point():
    c1 = scenes.c1_tiny(seed=0, noise_free=True)
    mo, mg = _build_pair(c1["map_points"], c1["voxel"], c1["cap"])
    og = far.default_options(conv_eps=1e-9)
    g = mg.gicp_register(c1["scan"], None, None, c1["T_init"], 2.0, 30, og)       # all covariances invalid -> SA fallback
    o = mo.gicp_register(c1["scan"], None, None, c1["T_init"], 2.0, 30, oracle.default_options(conv_eps=1e-9))
    dt, dr = _pose_err(g, o)
    assert dt < 1e-6 and dr < 1e-7
    dt, dr = _pose_err(g, dict(R=c1["T_gt"][0], t=c1["T_gt"][1]))
    assert dt < 1e-5 and g["chi2"] < 1e-6


def test_degenerate_and_max_iters():
    c1 = scenes.c1_tiny(seed=0)
    mo, mg = _build_pair(c1["map_points"], c1["voxel"], c1["cap"])
    far_away = (c1["scan"] + np.float32(500.0)).astype(np.float32)
    g = mg.gicp_register(far_away, None, None, c1["T_init"], 2.0, 30)
    assert g["status"] == far.ERR_DEGENERATE and g["n_inliers"] == 0 and g["iters"] == 1
    assert np.array_equal(g["R"], c1["T_init"][0]) and np.array_equal(g["t"], c1["T_init"][1])
    # max_iters = 2 stops early, not converged, pose equals the oracle's second iterate
    (cov_o, val_o), (cov_g, val_g) = _scan_cov(c1["scan"], c1["scan"], c1["voxel"], c1["cap"])
    o = mo.gicp_register(c1["scan"], cov_o, val_o, c1["T_init"], 2.0, 2)
    g = mg.gicp_register(c1["scan"], cov_g, val_g, c1["T_init"], 2.0, 2)
    assert g["iters"] == o["iters"] == 2 and g["converged"] == o["converged"] == 0
    dt, dr = _pose_err(g, o)
    assert dt < 1e-7 and dr < 1e-8
    # empty scan
    g = mg.gicp_register(np.zeros((0, 3), np.float32), None, None, c1["T_init"], 2.0, 5)
    assert g["status"] == far.ERR_DEGENERATE and g["n_inliers"] == 0


def test_c2_reduced_frame_end_to_end_device_chain():
    """A C2-shaped frame at reduced size (16 rings x 1024 azimuths, 200k-candidate map): voxelise -> Sigma_s ->
    register -> insert at the registered pose -> prune, chained on the device without host synchronisation,
    against the same steps on the oracle."""
    c2 = scenes.c2_single_frame(seed=1, n_map_candidates=200_000, map_radius=60.0, rings=16, azimuths=1024)
    v, cap, sigma = c2["voxel"], c2["cap"], c2["sigma"]
    mo, mg = _build_pair(c2["map_points"], v, cap)
    scan = c2["scan"]
    # oracle side
    ds_o, idx_o = oracle.voxelize(scan, v)
    lo = oracle.Map(v, cap); lo.insert(scan)
    cov_o, val_o = lo.knn_cov(ds_o, nthreads=8)
    o = mo.gicp_register(ds_o, cov_o, val_o, c2["T_init"], sigma, 30, nthreads=8)
    so = mo.insert(scan, pose=(o["R"], o["t"]), compute_cov=True)
    po = mo.prune(o["t"], 40.0)
    # device chain
    n = len(scan)
    d_scan = torch.as_tensor(scan).cuda()
    vox = far.Voxelizer(n)
    lg = far.Map(v, cap, 4 * n)
    d_cov = torch.empty((n, 6), dtype=torch.float32, device="cuda")
    d_val = torch.empty(n, dtype=torch.uint8, device="cuda")
    d_init = torch.frombuffer(bytearray(bytes(far.Pose.from_rt(c2["T_init"]))), dtype=torch.uint8).cuda()
    vox.enqueue(d_scan, v)
    lg.insert_enqueue(d_scan)
    lg.knn_cov(vox.out_xyz, out_cov=d_cov, out_valid=d_val, d_m=vox.n_out)
    res = mg.gicp_register_enqueue(vox.out_xyz, d_cov, d_val, None, sigma, 30, d_n=vox.n_out, d_init_pose=d_init)
    mg.insert_enqueue(d_scan, compute_cov=True, d_pose=res)            # the result struct starts with the pose
    mg.prune_enqueue(radius=40.0, d_pose=res)
    torch.cuda.synchronize()
    g = far.result_to_dict(far.GicpResult.from_buffer_copy(res.cpu().numpy().tobytes()))
    m = int(vox.n_out.item())
    assert m == len(idx_o) and np.array_equal(vox.out_index[:m].cpu().numpy(), idx_o)
    assert np.array_equal(d_val[:m].cpu().numpy(), val_o)
    assert g["status"] == o["status"] == 0 and g["iters"] == o["iters"] and g["n_inliers"] == o["n_inliers"]
    dt, dr = _pose_err(g, o)
    assert dt < 1e-4 and dr < 1e-5, (dt, dr)
    dt, dr = _pose_err(g, dict(R=c2["T_gt"][0], t=c2["T_gt"][1]))
    assert dt < 0.1 and dr < math.radians(0.5), (dt, dr)
    # the maps agree after insert + prune if the registered poses round the inserted points identically;
    # poses agree to ~1e-12, so compare structure exactly and coordinates to 1e-5 m
    eo, eg = mo.export(), mg.export()
    assert np.array_equal(eg["keys"], eo["keys"]) and np.array_equal(eg["counts"], eo["counts"])
    assert np.array_equal(eg["ids"], eo["ids"])
    assert np.abs(eg["xyz"] - eo["xyz"]).max() < 1e-5


def test_paper_parameters_v4_cap40_frame_matches_oracle():
    """The paper's own map parameters (v = 4 m, N_max = 40, k = 10): up to 27 x 40 = 1,080 candidates per
    query exercise the long candidate lists of the kNN / NN sweeps; Sigma_s, registration and the map update against
    the oracle on the reduced C2 scene."""
    c2 = scenes.c2_single_frame(seed=1, n_map_candidates=200_000, map_radius=60.0, rings=16, azimuths=1024)
    v, cap, sigma = 4.0, 40, c2["sigma"]
    mo, mg = _build_pair(c2["map_points"], v, cap)
    scan = c2["scan"]
    ds_o, idx_o = oracle.voxelize(scan, 1.0)
    ds_g, idx_g = far.voxelize(scan, 1.0)
    assert np.array_equal(idx_g.cpu().numpy(), idx_o)
    lo, lg = oracle.Map(v, cap), far.Map(v, cap, 1 << 14)
    lo.insert(scan); lg.insert(scan)
    cov_o, val_o = lo.knn_cov(ds_o, nthreads=8)
    cov_g, val_g = lg.knn_cov(ds_g)
    assert np.array_equal(val_g.cpu().numpy(), val_o) and val_o.mean() > 0.9
    cnt = mg.count27(ds_g).cpu().numpy()
    assert cnt.max() > 600                                  # the long lists really occur
    ids_o, d2_o = mo.nn(ds_o)
    ids_g, d2_g = mg.nn(ds_g)
    assert np.array_equal(ids_g.cpu().numpy().view(np.uint32), ids_o)
    assert np.array_equal(d2_g.cpu().numpy().view(np.uint32), d2_o.view(np.uint32))
    o = mo.gicp_register(ds_o, cov_o, val_o, c2["T_init"], sigma, 30, nthreads=8)
    g = mg.gicp_register(ds_g, cov_g, val_g, c2["T_init"], sigma, 30)
    assert g["status"] == o["status"] == 0 and g["iters"] == o["iters"] and g["n_inliers"] == o["n_inliers"]
    dt, dr = _pose_err(g, o)
    assert dt < 1e-4 and dr < 1e-5, (dt, dr)
    assert np.linalg.norm(g["H"] - o["H"]) <= 1e-4 * np.linalg.norm(o["H"])
    so = mo.insert(scan, pose=(o["R"], o["t"]), compute_cov=True)
    sg = mg.insert(scan, pose=(g["R"], g["t"]), compute_cov=True)
    assert sg == so
    eo, eg = mo.export(with_cov=True), mg.export(with_cov=True)
    assert np.array_equal(eg["keys"], eo["keys"]) and np.array_equal(eg["ids"], eo["ids"])
    assert np.array_equal(eg["cov_valid"], eo["cov_valid"])


def test_frontend_chain_equals_manual_chain_and_host_variant():
    """far_frontend_process (device scan) and far_frontend_process_host (host scan) give the oracle's frame."""
    c2 = scenes.c2_single_frame(seed=5, n_map_candidates=120_000, map_radius=50.0, rings=16, azimuths=512)
    v, cap, sigma = c2["voxel"], c2["cap"], c2["sigma"]
    scan = c2["scan"]
    mo = oracle.Map(v, cap)
    mo.insert(c2["map_points"], compute_cov=True)
    ds_o, _ = oracle.voxelize(scan, v)
    lo = oracle.Map(v, cap); lo.insert(scan)
    cov_o, val_o = lo.knn_cov(ds_o, nthreads=8)
    o = mo.gicp_register(ds_o, cov_o, val_o, c2["T_init"], sigma, 30, nthreads=8)
    mo.insert(scan, pose=(o["R"], o["t"]), compute_cov=True)
    mo.prune(o["t"], 35.0)
    eo = mo.export(with_cov=True)
    for host in (False, True):
        fe = far.Frontend(v, cap, 4 * len(c2["map_points"]), len(scan) + 7, prune_radius=35.0, max_iters=30)
        fe.map.insert(c2["map_points"], compute_cov=True)
        if host:
            g = fe.process_host(torch.as_tensor(scan).pin_memory(), c2["T_init"], sigma)
        else:
            d_res = torch.zeros(far.GICP_RESULT_BYTES, dtype=torch.uint8, device="cuda")
            fe.process_enqueue(torch.as_tensor(scan).cuda(), c2["T_init"], sigma, d_result=d_res)
            torch.cuda.synchronize()
            g = far.result_to_dict(far.GicpResult.from_buffer_copy(d_res.cpu().numpy().tobytes()))
        assert g["status"] == 0 and g["iters"] == o["iters"] and g["n_inliers"] == o["n_inliers"]
        dt, dr = _pose_err(g, o)
        assert dt < 1e-4 and dr < 1e-5, (dt, dr)
        eg = fe.map.export(with_cov=True)
        assert np.array_equal(eg["keys"], eo["keys"]) and np.array_equal(eg["ids"], eo["ids"])
        assert np.abs(eg["xyz"] - eo["xyz"]).max() < 1e-5
        assert np.array_equal(eg["cov_valid"], eo["cov_valid"])
        fe.close()


def test_frame_graph_replay_equals_stream_of_launches_and_oracle():
    """the frame as ONE CUDA graph.  Three frames of different sizes and poses through the same buffers: the
    first runs as a stream of launches, the second captures, the third replays; every frame's result and the final map
    equal those of the stream path (use_graph = 0) bit for bit and the oracle's within tolerance.  Per replayed frame the
    library launches no more kernels than the stream path does."""
    c2 = scenes.c2_single_frame(seed=6, n_map_candidates=100_000, map_radius=45.0, rings=16, azimuths=512)
    v, cap, sigma, scan = c2["voxel"], c2["cap"], c2["sigma"], c2["scan"]
    rng = np.random.default_rng(3)
    sizes = [len(scan), len(scan) - 1777, len(scan) - 31]
    poses = [c2["T_init"], scenes.perturb_pose(c2["T_gt"], 0.2, 1.0, rng), scenes.perturb_pose(c2["T_gt"], 0.1, 0.5, rng)]
    sig = [sigma, 1.0, 0.7]
    # oracle: three frames in a row on one map
    mo = oracle.Map(v, cap)
    mo.insert(c2["map_points"], compute_cov=True)
    res_o = []
    for n, T, sg in zip(sizes, poses, sig):
        s = scan[:n]
        ds_o, _ = oracle.voxelize(s, v)
        lo = oracle.Map(v, cap); lo.insert(s)
        cov_o, val_o = lo.knn_cov(ds_o, nthreads=8)
        o = mo.gicp_register(ds_o, cov_o, val_o, T, sg, 30, nthreads=8)
        mo.insert(s, pose=(o["R"], o["t"]), compute_cov=True)
        mo.prune(o["t"], 30.0)
        res_o.append(o)
    eo = mo.export(with_cov=True)
    outs = {}
    for use_graph in (False, True):
        fe = far.Frontend(v, cap, 4 * len(c2["map_points"]), len(scan), prune_radius=30.0, max_iters=30, use_graph=use_graph)
        fe.map.insert(c2["map_points"], compute_cov=True)
        buf = torch.zeros((len(scan), 3), dtype=torch.float32, device="cuda")      # ONE scan buffer, as a driver would keep
        d_res = torch.zeros(far.GICP_RESULT_BYTES, dtype=torch.uint8, device="cuda")
        rs, launches = [], []
        for n, T, sg in zip(sizes, poses, sig):
            buf[:n] = torch.as_tensor(scan[:n]).cuda()
            l0 = far.launch_count()
            rc = far.lib().far_frontend_process(fe._h, buf.data_ptr(), n, 3, far.C.byref(far.Pose.from_rt(T)), sg, d_res.data_ptr(),
                                                torch.cuda.current_stream().cuda_stream)
            assert rc == far.OK
            launches.append(far.launch_count() - l0)
            torch.cuda.synchronize()
            rs.append(d_res.cpu().numpy().tobytes())
        assert fe.graph_state() == (1 if use_graph else 0)
        assert launches[2] == launches[0] and launches[0] <= 20
        outs[use_graph] = (rs, fe.map.export(with_cov=True), fe.map.stats())
        fe.close()
    (ra, ea, sa), (rb, eb, sb) = outs[False], outs[True]
    assert ra == rb                                           # far_gicp_result_t bytes of every frame
    for k in ("keys", "counts", "ids", "xyz", "cov", "cov_valid"):
        assert np.array_equal(ea[k].view(np.uint8), eb[k].view(np.uint8)), k
    assert sa == sb
    for raw, o in zip(rb, res_o):
        g = far.result_to_dict(far.GicpResult.from_buffer_copy(raw))
        assert g["status"] == 0 and g["iters"] == o["iters"] and g["n_inliers"] == o["n_inliers"]
        dt, dr = _pose_err(g, o)
        assert dt < 1e-4 and dr < 1e-5, (dt, dr)
    assert np.array_equal(eb["keys"], eo["keys"]) and np.array_equal(eb["ids"], eo["ids"])
    assert np.abs(eb["xyz"] - eo["xyz"]).max() < 1e-5
    assert np.array_equal(eb["cov_valid"], eo["cov_valid"])


def test_empty_frame_without_a_scan_pointer_is_a_frame_like_any_other():
    """far_frontend_process accepts n == 0 with a NULL scan (far.h: "(n > 0 && !d_scan)" is the error).  The frame runs its
    whole chain on zero points: the registration reports FAR_ERR_DEGENERATE with the initial pose (fewer than 6 inliers,
    PAPER.md:84-100 has nothing to solve), the map is untouched, and neither the stream path nor the captured graph is
    disturbed -- the frames after it give the bytes they give without the empty frame in between."""
    c1 = scenes.c1_tiny(seed=0)
    v, cap, scan = c1["voxel"], c1["cap"], c1["scan"]
    st = torch.cuda.current_stream().cuda_stream
    runs = {}
    for with_empty in (False, True):
        fe = far.Frontend(v, cap, 1 << 14, len(scan), ds_voxel=v, prune_radius=50.0, max_iters=c1["max_iters"])
        fe.map.insert(c1["map_points"], compute_cov=True)
        buf = torch.as_tensor(scan).cuda()
        d_res = torch.zeros(far.GICP_RESULT_BYTES, dtype=torch.uint8, device="cuda")
        po = far.Pose.from_rt(c1["T_init"])
        frames = []
        for k in range(5):
            if with_empty and k in (0, 3):          # before anything ran, and after the graph was captured
                before = fe.map.export(with_cov=True)
                rc = far.lib().far_frontend_process(fe._h, None, 0, 3, far.C.byref(po), c1["sigma"], d_res.data_ptr(), st)
                assert rc == far.OK
                torch.cuda.synchronize()
                g = far.result_to_dict(far.GicpResult.from_buffer_copy(d_res.cpu().numpy().tobytes()))
                assert g["status"] == far.ERR_DEGENERATE and g["n_inliers"] == 0
                assert np.array_equal(g["R"], np.asarray(c1["T_init"][0])) and np.array_equal(g["t"], np.asarray(c1["T_init"][1]))
                after = fe.map.export(with_cov=True)
                for key in ("keys", "counts", "ids", "xyz", "cov", "cov_valid"):
                    assert np.array_equal(before[key].view(np.uint8), after[key].view(np.uint8)), key
                assert fe.graph_state() >= 0
            rc = far.lib().far_frontend_process(fe._h, buf.data_ptr(), len(scan), 3, far.C.byref(po), c1["sigma"], d_res.data_ptr(), st)
            assert rc == far.OK
            torch.cuda.synchronize()
            frames.append(d_res.cpu().numpy().tobytes())
        assert fe.graph_state() == 1
        runs[with_empty] = (frames, fe.map.export(with_cov=True))
        fe.close()
    assert runs[False][0] == runs[True][0]
    for key in ("keys", "counts", "ids", "xyz", "cov", "cov_valid"):
        assert np.array_equal(runs[False][1][key].view(np.uint8), runs[True][1][key].view(np.uint8)), key
    first = far.result_to_dict(far.GicpResult.from_buffer_copy(runs[True][0][0]))
    assert first["status"] == 0 and first["n_inliers"] > 100


def test_ten_thousand_registrations_are_bitwise_reproducible():
    """The reduction is a fixed-order sum of tagged words (far_gicp.cu): 10,000 back-to-back registrations, two maps
    alternating (each with its own scratch and launch sequence), no host synchronisation in between -- every
    far_gicp_result_t must be byte-identical to the first one of its map.  A torn or stale tagged word, a reused tag or a
    summation order that depends on arrival would show up here."""
    c1 = scenes.c1_tiny(seed=0)
    v, cap = c1["voxel"], c1["cap"]
    maps, scans, poses = [], [], []
    for j in range(2):
        m = far.Map(v, cap, 1 << 14, with_cov=True)
        m.insert(c1["map_points"], compute_cov=True)
        lm = far.Map(v, cap, 1 << 13)
        sc = c1["scan"] if j == 0 else c1["scan"][::-1].copy()
        lm.insert(sc)
        ds = torch.as_tensor(sc).cuda()
        cov, val = lm.knn_cov(ds)
        maps.append(m); scans.append((ds, cov, val))
        poses.append(c1["T_init"] if j == 0 else scenes.perturb_pose(c1["T_init"], 0.05, 0.5, np.random.default_rng(1)))
    n_rep = 5000
    out = torch.zeros((2, n_rep, far.GICP_RESULT_BYTES), dtype=torch.uint8, device="cuda")
    for r in range(n_rep):
        for j in range(2):
            ds, cov, val = scans[j]
            maps[j].gicp_register_enqueue(ds, cov, val, poses[j], c1["sigma"], 30, d_result=out[j, r])
    torch.cuda.synchronize()
    h = out.cpu().numpy()
    for j in range(2):
        first = far.result_to_dict(far.GicpResult.from_buffer_copy(h[j, 0].tobytes()))
        assert first["status"] == 0 and first["iters"] > 3
        assert (h[j] == h[j, 0]).all(), np.nonzero((h[j] != h[j, 0]).any(axis=1))[0][:5]
    for m in maps:
        m.close()
