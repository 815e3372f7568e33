"""The host-side Sensor Fusion module of the product (far_ekf_*, C++ FP64) against the NumPy oracle
(oracle/ekf.py) on seeded synthetic IMU + delayed LiDAR measurements.  Host-only: runs without a GPU."""
import numpy as np
import pytest

import far_scenes as scenes
import paper_2606_26010_b200 as far
from oracle import ekf as oekf


def test_model_step_and_analytic_jacobian_match_oracle_central_differences():
    rng = np.random.default_rng(0)
    for _ in range(25):
        x = np.r_[rng.normal(0, 50, 3), rng.uniform(-0.6, 0.6, 2), rng.uniform(-3, 3), rng.normal(0, 20, 3)]
        u = np.r_[rng.normal(0, 3, 3) + [0, 0, 9.8], rng.normal(0, 0.5, 3)]
        xn, F = far.ekf_model(x, u, 0.01)
        assert np.allclose(xn, oekf.f(x, u, 0.01), rtol=0, atol=1e-12)
        assert np.allclose(F, oekf.jacobian_f(x, u, 0.01), atol=2e-8)


def test_lidar_velocity_eq7_matches_oracle():
    rng = np.random.default_rng(1)
    T0 = scenes.pose_from_rpy_t(0.02, -0.01, 0.7, rng.normal(0, 10, 3))
    T1 = scenes.pose_from_rpy_t(0.01, 0.0, 0.72, T0[1] + [5.0, 4.0, 0.1])
    assert np.allclose(far.lidar_velocity(T1, T0, 0.1), oekf.lidar_velocity(T1[0], T1[1], T0[1], 0.1), atol=1e-12)


def _trajectory(seed, n):
    """IMU samples of a car accelerating through a bend (specific force + rates, with noise)"""
    rng = np.random.default_rng(seed)
    k = np.arange(n)
    w = np.stack([0.02 * np.sin(k / 40), 0.01 * np.cos(k / 55), 0.3 * np.sin(k / 150)], axis=1)
    a = np.stack([2.0 * np.cos(k / 90), 30.0 * w[:, 2], np.full(n, oekf.G0)], axis=1)
    return a + rng.normal(0, 0.05, a.shape), w + rng.normal(0, 0.002, w.shape), rng


@pytest.mark.parametrize("n_up,with_ref", [(1, False), (10, False), (5, True)])
def test_filter_matches_oracle_with_delayed_upsampled_lidar(n_up, with_ref):
    n = 400
    a, w, rng = _trajectory(3 + n_up, n)
    x0 = np.r_[0, 0, 0, 0, 0, 0.3, 30.0, 0, 0]
    P0 = np.r_[[0.1] * 3, [1e-3] * 3, [0.05] * 3]
    Q = np.r_[[1e-6] * 3, [1e-7] * 3, [1e-4] * 3]
    ab, wb = np.array([0.02, -0.01, 0.03]), np.array([1e-3, -2e-3, 5e-4])
    g = far.Ekf(x0, P0, Q, dt=0.01, n_up=n_up, accel_bias=ab, gyro_bias=wb)
    o = oekf.Ekf(x0, np.diag(P0), np.diag(Q), dt=0.01, n_up=n_up, a_b=ab, w_b=wb)
    m = 11 if with_ref else 9
    Rd = np.r_[[1e-3] * 3, [1e-5] * 3, ([1e-4] * 2 if with_ref else []), [1e-2] * 3]
    for k in range(n):
        kg = g.predict(a[k], w[k])
        o.predict(np.r_[a[k], w[k]])
        assert kg == o.k
        if k % 10 == 9 and k > 20:
            # a LiDAR pose taken 6 cycles ago (60 ms latency) arrives now
            s = o.k - 6
            xs = o.history[s] + np.r_[rng.normal(0, 0.03, 3), rng.normal(0, 0.003, 3), rng.normal(0, 0.1, 3)]
            T_L = scenes.pose_from_rpy_t(xs[3], xs[4], xs[5], xs[0:3])
            ref = xs[3:5] + rng.normal(0, 0.01, 2) if with_ref else None
            g.push_lidar(T_L, xs[6:9], Rd, s, theta_ref=ref)
            z = np.r_[xs[0:6], (ref if with_ref else []), xs[6:9]]
            assert len(z) == m
            o.push_measurement(z, np.diag(Rd), s, with_ref=with_ref)
        xg, Pg, _ = g.state()
        assert np.allclose(xg, o.x, atol=1e-7), k
        assert np.allclose(Pg, o.P, rtol=1e-5, atol=2e-9), k      # the oracle differentiates f numerically (1e-9 in F)
    R, t = g.pose()
    assert np.allclose(R, oekf.rot(o.x[3:6]), atol=1e-8) and np.allclose(t, o.x[0:3], atol=1e-7)


def test_velocity_history_feeds_the_motion_fit():
    n = 60
    a, w, _ = _trajectory(9, n)
    wb = np.array([1e-3, 0, -1e-3])
    g = far.Ekf(np.r_[0, 0, 0, 0, 0, 0, 25.0, 0, 0], [1e-2] * 9, [1e-6] * 9, dt=0.01, gyro_bias=wb)
    xs = []
    for k in range(n):
        g.predict(a[k], w[k])
        xs.append(g.state()[0])
    t, v = g.velocity_history(20)
    assert len(t) == 20 and np.allclose(t, np.arange(41, 61) * 0.01)
    assert np.allclose(v[:, :3], np.array(xs)[40:60, 6:9]) and np.allclose(v[:, 3:], w[40:60] - wb)
    a_fit, b_fit = far.motion_fit(t, v, t[-1])
    assert np.isfinite(a_fit).all() and abs(a_fit[0] - xs[-1][6]) < 0.05


def test_push_rejects_measurements_outside_the_history():
    g = far.Ekf(np.zeros(9), [1.0] * 9, [0.0] * 9)
    g.predict([0, 0, oekf.G0], [0, 0, 0])
    T = scenes.pose_identity()
    with pytest.raises(far.FarError):
        g.push_lidar(T, [0, 0, 0], [1.0] * 9, cycle_s=5)          # the future
    with pytest.raises(far.FarError):
        g.push_lidar(T, [0, 0, 0], [0.0] * 9, cycle_s=0)          # non-positive variance


def test_covariance_propagates_with_the_jacobian_of_the_step_actually_taken():
    """Pin independent of the oracle (R18): with non-zero biases, P after one cycle must be F P F^T + Q with F the finite
    difference of the PRODUCT's own state step (same inputs, perturbed states).  A Jacobian evaluated at the raw gyro rate
    in the E(theta) w block -- the step uses w_m - w_b there -- fails this."""
    rng = np.random.default_rng(12)
    x0 = np.r_[1.0, -2.0, 0.5, 0.05, -0.08, 0.7, 25.0, 0.4, -0.2]
    P0 = np.r_[[0.2] * 3, [2e-3] * 3, [0.1] * 3]
    Q = np.r_[[1e-6] * 3, [1e-7] * 3, [1e-4] * 3]
    ab, wb = np.array([0.3, -0.2, 0.1]), np.array([0.2, -0.3, 0.25])          # large gyro bias: the two Jacobians differ visibly
    a_m, w_m = np.array([0.5, 1.0, 9.6]), np.array([0.3, 0.2, 0.6])
    dt = 0.01

    def step(x):
        e = far.Ekf(x, P0, Q, dt=dt, accel_bias=ab, gyro_bias=wb)
        e.predict(a_m, w_m)
        return e.state()

    xn, Pn, _ = step(x0)
    F = np.zeros((9, 9))
    h = 1e-6
    for j in range(9):
        d = np.zeros(9); d[j] = h
        F[:, j] = (step(x0 + d)[0] - step(x0 - d)[0]) / (2 * h)
    want = F @ np.diag(P0) @ F.T + np.diag(Q)
    assert np.allclose(Pn, want, rtol=1e-6, atol=1e-10)
    # and it is not the raw-rate Jacobian: that one differs in the attitude block by dt * d(E(theta) w_b)/d(theta)
    _, F_raw = far.ekf_model(x0, np.r_[a_m, w_m], dt)
    assert np.abs(F_raw - F).max() > 1e-4
    # the oracle takes the same Jacobian
    assert np.allclose(oekf.jacobian_f(x0, np.r_[a_m, w_m], dt, ab, wb), F, atol=1e-7)
