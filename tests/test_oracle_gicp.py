"""Pins for the oracle's kNN covariance (A7, Eq. 1) and GICP linearisation / registration (A8-A10)."""
import math

import numpy as np
import pytest
from scipy.linalg import expm

import far_scenes as fs
import oracle
from helpers import hat, load_golden, np_voxel_index, rot_angle, twist_matrix


def sym(c6):
    c = np.asarray(c6, dtype=np.float64)
    return np.array([[c[0], c[1], c[2]], [c[1], c[3], c[4]], [c[2], c[4], c[5]]])


# ----------------------------------------------------------------------------- A7 covariance
def test_cov_eq1_closed_form_golden():
    g = load_golden("cov_eq1_closed_form.json")
    # 10 points whose biased sample covariance is exactly diag(0.1, 0.1, 0): +-a on x (4 pts), +-a on y (4), 2 at 0
    a = math.sqrt(0.1 * 10 / 4)
    pts = np.array([[a, 0, 0], [-a, 0, 0], [a, 0, 0], [-a, 0, 0], [0, a, 0], [0, -a, 0], [0, a, 0], [0, -a, 0],
                    [0, 0, 0], [0, 0, 0]], dtype=np.float64)
    S = sym(oracle.cov_from_points(pts.astype(np.float32), g["eps"]))
    ev = np.sort(np.linalg.eigvalsh(S))
    assert ev == pytest.approx(sorted(g["eig_sigma"]), rel=1e-6)


def test_cov_eq1_properties_random():
    rng = np.random.default_rng(0)
    for _ in range(50):
        pts = (rng.normal(size=(10, 3)) * rng.uniform(0.01, 2.0, size=3) + rng.uniform(-100, 100, size=3)).astype(np.float32)
        S = sym(oracle.cov_from_points(pts, 1e-3))
        assert np.allclose(S, S.T)
        assert np.linalg.eigvalsh(S).min() > 0                       # SPD
        assert np.linalg.norm(np.linalg.inv(S), "fro") == pytest.approx(1.0, abs=1e-9)    # ||Sigma^-1||_F = 1
        # explicit double inversion of Eq. 1 with library routines
        Shat = np.cov(pts.astype(np.float64).T, bias=True)             # 1/k (reading R7)
        Cm = Shat + 1e-3 * np.eye(3)
        Ci = np.linalg.inv(Cm)
        want = np.linalg.inv(Ci / np.linalg.norm(Ci, "fro"))
        assert np.allclose(S, want, rtol=1e-8, atol=1e-10)


def test_cov_plane_normal_is_smallest_eigenvector():
    rng = np.random.default_rng(1)
    n = np.array([1.0, 2.0, -0.5])
    n /= np.linalg.norm(n)
    e1 = np.cross(n, [0, 0, 1.0]); e1 /= np.linalg.norm(e1)
    e2 = np.cross(n, e1)
    uv = rng.uniform(-1, 1, size=(10, 2))
    pts = (uv[:, :1] * e1 + uv[:, 1:] * e2).astype(np.float32)
    S = sym(oracle.cov_from_points(pts, 1e-3))
    w, V = np.linalg.eigh(S)
    assert abs(abs(V[:, 0] @ n) - 1.0) < 1e-5
    assert w[0] == pytest.approx(1.0, abs=2e-3)        # ~1.0001-ish: the regularised normal direction
    assert w[1] > 50


def _c1(noise_free=False):
    c1 = fs.c1_tiny(noise_free=noise_free)
    m = oracle.Map(c1["voxel"], c1["cap"])
    m.insert(c1["map_points"], compute_cov=True)
    sm = oracle.Map(c1["voxel"], c1["cap"])
    sm.insert(c1["scan"])
    cov_s, valid_s = sm.knn_cov(c1["scan"])
    return c1, m, cov_s, valid_s


def test_knn_ids_vs_numpy_bruteforce_and_cov():
    c1, m, _, _ = _c1()
    exp = m.export(with_cov=True)
    sel = np.concatenate([np.arange(c) + v * m.cap for v, c in enumerate(exp["counts"])])
    sx = exp["xyz"].reshape(-1, 3)[sel]
    sid = exp["ids"].reshape(-1)[sel]
    mk = np_voxel_index(sx, c1["voxel"])
    q = c1["scan"][:150]
    ids, d2 = m.knn(q, 10)
    cov, valid = m.knn_cov(q)
    qk = np_voxel_index(q, c1["voxel"])
    n_invalid = 0
    for i in range(len(q)):
        adj = np.all(np.abs(mk - qk[i]) <= 1, axis=1)
        d = q[i].astype(np.float64) - sx[adj].astype(np.float64)
        dd = (d[:, 0] * d[:, 0] + d[:, 1] * d[:, 1]) + d[:, 2] * d[:, 2]
        cid = sid[adj]
        order = np.lexsort((cid, dd))[:10]
        k = len(order)
        assert np.array_equal(ids[i, :k], cid[order])
        assert np.array_equal(d2[i, :k], dd[order])
        if k < 10:
            assert valid[i] == 0 and np.array_equal(cov[i], [1, 0, 0, 1, 0, 1])
            assert (ids[i, k:] == oracle.NO_ID).all()
            n_invalid += 1
        else:
            assert valid[i] == 1
            nb = sx[adj][order].astype(np.float64)
            Cm = np.cov(nb.T, bias=True) + 1e-3 * np.eye(3)
            want = np.linalg.norm(np.linalg.inv(Cm), "fro") * Cm
            assert np.allclose(sym(cov[i]), want, rtol=2e-6)
    # stored covariances of map points: the point itself is its own first neighbour (d2 = 0)
    ids0, d20 = m.knn(sx[:50], 1)
    assert np.array_equal(ids0[:, 0], sid[:50]) and (d20 == 0).all()


def test_knn_cov_invalid_when_fewer_than_k():
    m = oracle.Map(0.5, 20)
    m.insert(np.random.default_rng(2).uniform(0, 0.4, size=(9, 3)).astype(np.float32), compute_cov=True)
    cov, valid = m.knn_cov(np.array([[0.2, 0.2, 0.2]], dtype=np.float32))
    assert valid[0] == 0 and cov[0].tolist() == [1, 0, 0, 1, 0, 1]
    assert m.export(with_cov=True)["cov_valid"].sum() == 0
    m.insert(np.array([[0.1, 0.1, 0.1]], dtype=np.float32), compute_cov=True)
    e = m.export(with_cov=True)
    # only the ADDED point gets a covariance; existing ones stay unchanged
    assert e["cov_valid"].sum() == 1 and e["cov_valid"][0, 9] == 1


# ----------------------------------------------------------------------------- robust weights, Exp, threshold
def test_robust_weight_golden():
    g = load_golden("robust_weights.json")
    assert oracle.robust_weight(oracle.KERNEL_CAUCHY, g["e2"], g["kappa"]) == pytest.approx(g["cauchy"], rel=1e-12)
    assert oracle.robust_weight(oracle.KERNEL_GEMAN_MCCLURE, g["e2"], g["kappa"]) == pytest.approx(g["geman_mcclure"], rel=1e-12)
    assert oracle.robust_weight(oracle.KERNEL_NONE, g["e2"], g["kappa"]) == 1.0
    # Cauchy weight is rho'(e)/e of Eq. 5: finite-difference the printed rho
    k, e = 0.7, 0.9
    rho = lambda x: k * k / 2 * math.log(1 + (x / k) ** 2)
    h = 1e-6
    assert oracle.robust_weight(oracle.KERNEL_CAUCHY, e * e, k) == pytest.approx((rho(e + h) - rho(e - h)) / (2 * h) / e, rel=1e-6)


def test_se3_exp_vs_scipy_expm():
    rng = np.random.default_rng(3)
    for scale in [1e-12, 1e-9, 1e-6, 1e-3, 0.1, 1.0, 3.0]:
        d = rng.normal(size=6) * scale
        R, t = oracle.se3_exp(d)
        X = expm(twist_matrix(d))
        assert np.allclose(R, X[:3, :3], atol=1e-13) and np.allclose(t, X[:3, 3], atol=1e-13 * max(1, scale))
        assert np.allclose(R @ R.T, np.eye(3), atol=1e-13)


def test_adaptive_threshold_closed_form():
    th = oracle.AdaptiveThreshold(sigma0=2.0, min_motion=0.1, max_range=100.0)
    assert th.sigma() == 2.0
    P = fs.pose_from_rpy_t(0, 0, 0.3, [1, 2, 3])
    dT = fs.pose_from_rpy_t(0, 0, 0.01, [0.3, 0.0, 0.4])
    th.update(P, fs.pose_compose(P, dT))
    want = 0.5 + 2 * 100.0 * math.sin(0.005)
    assert th.sigma() == pytest.approx(want, rel=1e-9)
    small = fs.pose_from_rpy_t(0, 0, 0.0, [0.05, 0, 0])
    th.update(P, fs.pose_compose(P, small))            # delta <= min_motion: not recorded
    assert th.sigma() == pytest.approx(want, rel=1e-9)
    dT2 = fs.pose_from_rpy_t(0, 0, 0.0, [1.0, 0, 0])
    th.update(P, fs.pose_compose(P, dT2))
    assert th.sigma() == pytest.approx(math.sqrt((want ** 2 + 1.0) / 2), rel=1e-9)


# ----------------------------------------------------------------------------- A8-A10 linearisation
def test_single_correspondence_golden():
    g = load_golden("gicp_single_correspondence.json")
    m = oracle.Map(0.5, 20)
    m.insert(np.array([g["r"]], dtype=np.float32))
    opts = oracle.default_options(kernel=oracle.KERNEL_NONE)
    res = m.gicp_linearize(np.array([g["p"]], dtype=np.float32), None, None, fs.pose_identity(), 2.0, opts)
    assert res["n_inliers"] == 1
    assert np.allclose(res["b"], g["b"], atol=1e-8)       # r = (1,0,0.1) is not exact in fp32
    assert np.allclose(res["H"], np.array(g["H"], dtype=float), atol=1e-12)
    assert np.linalg.matrix_rank(res["H"]) == 3


@pytest.mark.parametrize("kernel", [oracle.KERNEL_CAUCHY, oracle.KERNEL_GEMAN_MCCLURE, oracle.KERNEL_NONE])
def test_linearise_H_psd_and_b_is_gradient(kernel):
    c1, m, cov_s, valid_s = _c1()
    opts = oracle.default_options(kernel=kernel)
    T = fs.pose_from_rpy_t(0.01, -0.02, 0.05, [0.1, 0.05, -0.03])
    res = m.gicp_linearize(c1["scan"], cov_s, valid_s, T, 2.0, opts)
    H, b = res["H"], res["b"]
    assert np.allclose(H, H.T, rtol=1e-12, atol=1e-9)
    assert np.linalg.eigvalsh(0.5 * (H + H.T)).min() > 0
    cor = m.gicp_correspondences(c1["scan"], cov_s, valid_s, T, 2.0, opts)
    u = cor["used"]
    assert u.sum() == res["n_inliers"] > 900
    # both branches exercised: full GICP (M != I) and the sparsity-aware fallback (M == I)
    isI = np.all(np.isclose(cor["M"][u], np.eye(3)), axis=(1, 2))
    assert isI.any() and (~isI).any()
    p, r, M, w = cor["p"][u], cor["r"][u], cor["M"][u], cor["w"][u]

    def cost(delta):       # 1/2 sum w d^T M d with w, M frozen and p -> Exp(delta) p
        X = expm(twist_matrix(delta))
        d = r - (p @ X[:3, :3].T + X[:3, 3])
        return 0.5 * np.sum(w * np.einsum("ni,nij,nj->n", d, M, d))
    h = 1e-6
    grad = np.array([(cost(h * e) - cost(-h * e)) / (2 * h) for e in np.eye(6)])
    assert np.allclose(b, grad, rtol=1e-6, atol=1e-6 * np.abs(grad).max())
    # Gauss-Newton Hessian: second difference of the frozen-weight cost along random directions (first-order J)
    chi2 = np.sum(w * np.einsum("ni,nij,nj->n", r - p, M, r - p))
    assert res["chi2"] == pytest.approx(chi2, rel=1e-12)
    # explicit normal equations in NumPy
    J = np.zeros((len(p), 3, 6))
    J[:, :, :3] = -np.eye(3)
    J[:, :, 3:] = np.array([hat(x) for x in p])
    Hn = np.einsum("n,nia,nij,njb->ab", w, J, M, J)
    bn = np.einsum("n,nia,nij,nj->a", w, J, M, r - p)
    assert np.allclose(H, Hn, rtol=1e-10) and np.allclose(b, bn, rtol=1e-10, atol=1e-10)


def test_M_matches_numpy_inverse_and_gate():
    c1, m, cov_s, valid_s = _c1()
    T = fs.pose_from_rpy_t(0.0, 0.0, 0.03, [0.1, 0.0, 0.0])
    opts = oracle.default_options()
    cor = m.gicp_correspondences(c1["scan"], cov_s, valid_s, T, 2.0, opts)
    exp = m.export(with_cov=True)
    idmap = {}
    for v in range(len(exp["keys"])):
        for j in range(exp["counts"][v]):
            idmap[int(exp["ids"][v, j])] = (exp["cov"][v, j], exp["cov_valid"][v, j])
    R = T[0]
    checked = 0
    for i in np.nonzero(cor["used"])[0][:200]:
        cr, vr = idmap[int(cor["id"][i])]
        if vr and valid_s[i]:
            want = np.linalg.inv(sym(cr) + R @ sym(cov_s[i]) @ R.T)
            assert np.allclose(cor["M"][i], want, rtol=1e-9)
            checked += 1
        else:
            assert np.array_equal(cor["M"][i], np.eye(3))          # SA fallback
    assert checked > 50
    # the gate: sigma so small that tau = 3 sigma rejects everything farther than 3 cm
    cor2 = m.gicp_correspondences(c1["scan"], cov_s, valid_s, T, 0.01, opts)
    ids, d2 = m.nn(fs.pose_apply(T, c1["scan"]))
    # note: pose_apply uses a matmul; the oracle's fixed-order transform can differ in the last bit, so compare counts loosely
    assert abs(int(cor2["used"].sum()) - int((d2 <= 0.03 ** 2).sum())) <= 3


def test_point_to_point_fixed_correspondences_equals_kabsch():
    """All covariances invalid + kernel NONE = point-to-point ICP; with correspondences that do not change, the
    converged pose is the Kabsch/SVD closed form."""
    rng = np.random.default_rng(5)
    mp = rng.uniform(-4, 4, size=(60, 3)).astype(np.float32) * np.array([1, 1, 0.3], dtype=np.float32)
    # well separated points so NN correspondences are stable for a small motion
    m = oracle.Map(4.0, 40)
    m.insert(mp)
    T_gt = fs.pose_from_rpy_t(0.01, -0.015, 0.02, [0.03, -0.02, 0.01])
    scan = (fs.pose_apply(fs.pose_inverse(T_gt), mp).astype(np.float64) + rng.normal(0, 0.005, size=mp.shape)).astype(np.float32)
    opts = oracle.default_options(kernel=oracle.KERNEL_NONE, conv_eps=1e-12)
    res = m.gicp_register(scan, None, None, fs.pose_identity(), 2.0, 50, opts)
    ids, _ = m.nn(fs.pose_apply((res["R"], res["t"]), scan))
    assert np.array_equal(ids, np.arange(60))
    A = scan.astype(np.float64); B = mp.astype(np.float64)
    ca, cb = A.mean(0), B.mean(0)
    U, _, Vt = np.linalg.svd((A - ca).T @ (B - cb))
    D = np.diag([1, 1, np.sign(np.linalg.det(Vt.T @ U.T))])
    Rk = Vt.T @ D @ U.T
    tk = cb - Rk @ ca
    assert np.allclose(res["R"], Rk, atol=1e-7) and np.allclose(res["t"], tk, atol=1e-7)


@pytest.mark.parametrize("kernel", [oracle.KERNEL_CAUCHY, oracle.KERNEL_GEMAN_MCCLURE])
def test_noise_free_recovery(kernel):
    c1, m, cov_s, valid_s = _c1(noise_free=True)
    opts = oracle.default_options(kernel=kernel, conv_eps=1e-9)
    res = m.gicp_register(c1["scan"], cov_s, valid_s, c1["T_init"], 2.0, 30, opts)
    assert res["status"] == 0 and res["converged"] == 1
    R, t = c1["T_gt"]
    assert np.linalg.norm(res["t"] - t) < 1e-5            # fp32 scan coordinates: ~1e-7 m rounding
    assert rot_angle(res["R"].T @ R) < 1e-6
    assert res["chi2"] < 1e-6


def test_c1_registration_converges():
    c1, m, cov_s, valid_s = _c1()
    for eps, max_it in [(5e-3, 12), (1e-6, 30)]:
        res = m.gicp_register(c1["scan"], cov_s, valid_s, c1["T_init"], 2.0, 30, oracle.default_options(conv_eps=eps))
        assert res["converged"] == 1 and res["iters"] <= max_it and res["n_inliers"] == 1024
        R, t = c1["T_gt"]
        assert np.linalg.norm(res["t"] - t) < 5e-3 and rot_angle(res["R"].T @ R) < 2e-3
    # multi-threaded linearisation sums in index order: identical bits
    a = m.gicp_linearize(c1["scan"], cov_s, valid_s, c1["T_init"], 2.0, None, nthreads=1)
    b = m.gicp_linearize(c1["scan"], cov_s, valid_s, c1["T_init"], 2.0, None, nthreads=4)
    assert np.array_equal(a["H"], b["H"]) and np.array_equal(a["b"], b["b"])


def test_degenerate_returns_init_pose():
    m = oracle.Map(0.5, 20)
    m.insert(np.array([[0, 0, 0], [1, 0, 0]], dtype=np.float32))
    T0 = fs.pose_from_rpy_t(0, 0, 0.1, [0.01, 0, 0])
    res = m.gicp_register(np.array([[0, 0, 0.05], [1, 0, 0.05]], dtype=np.float32), None, None, T0, 2.0, 5, None)
    assert res["status"] == oracle.ERR_DEGENERATE
    assert np.array_equal(res["R"], T0[0]) and np.array_equal(res["t"], T0[1])
