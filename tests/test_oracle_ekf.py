"""Pins for the oracle's kinematic EKF (Eq. 7-11; R18-R20): closed forms of the motion
model, finite-difference-free identities of the Kalman update, and textbook linear-Gaussian results."""
import numpy as np
import pytest
from scipy.spatial.transform import Rotation

from oracle import ekf


def test_rotation_and_euler_rates_match_scipy_and_definition():
    rng = np.random.default_rng(0)
    for _ in range(20):
        th = rng.uniform(-1.2, 1.2, 3)
        assert np.allclose(ekf.rot(th), Rotation.from_euler("ZYX", th[::-1]).as_matrix(), atol=1e-14)
        # E(theta) w = d theta / dt  <=>  d R / dt = R [w]x : check with a small body rotation
        w = rng.normal(0, 1, 3)
        h = 1e-6
        th2 = th + ekf.euler_rates(th) @ w * h
        dR = (ekf.rot(th2) - ekf.rot(th)) / h
        assert np.allclose(dR, ekf.rot(th) @ ekf.hat(w), atol=1e-5)


def test_motion_model_static_and_level_is_a_fixed_point():
    # at rest, any attitude: the accelerometer reads -g(theta) (specific force), the state must not move
    for th in ([0, 0, 0], [0.1, -0.2, 1.0]):
        x = np.r_[[1.0, 2.0, 3.0], th, [0, 0, 0]]
        a_m = -ekf.rot(th).T @ np.array([0, 0, -ekf.G0])
        x1 = ekf.f(x, np.r_[a_m, 0, 0, 0], 0.01)
        assert np.allclose(x1, x, atol=1e-15)


def test_motion_model_straight_line_and_circle_closed_forms():
    dt, n = 0.001, 2000
    # straight: constant body velocity, heading 0.5 rad
    x = np.r_[0, 0, 0, 0, 0, 0.5, 20.0, 0, 0]
    a_m = np.array([0, 0, ekf.G0])
    for _ in range(n):
        x = ekf.f(x, np.r_[a_m, 0, 0, 0], dt)
    assert np.allclose(x[:3], 20.0 * n * dt * np.array([np.cos(0.5), np.sin(0.5), 0]), atol=1e-9)
    # circle: speed v, yaw rate w; body-frame velocity stays (v,0,0) only if the accelerometer reads the centripetal
    # acceleration a_y = v w (that is what -[w]x v + a_m cancels); radius v/w
    v, w = 30.0, 0.5
    x = np.r_[0, 0, 0, 0, 0, 0, v, 0, 0]
    u = np.r_[0, v * w, ekf.G0, 0, 0, w]
    for _ in range(n):
        x = ekf.f(x, u, dt)
    T = n * dt
    assert np.allclose(x[6:9], [v, 0, 0], atol=1e-9)
    assert abs(x[5] - w * T) < 1e-12
    want = np.array([v / w * np.sin(w * T), v / w * (1 - np.cos(w * T)), 0])
    assert np.linalg.norm(x[:3] - want) < 0.02          # explicit Euler: O(dt) position error (v w dt T / 2 = 0.015)


def test_lidar_velocity_eq7():
    R = ekf.rot([0, 0, np.pi / 2])
    v = ekf.lidar_velocity(R, [0, 7.0, 0], [0, 0, 0], 0.1)     # moving +y in the map = forward for a sensor yawed 90 deg
    assert np.allclose(v, [70.0, 0, 0], atol=1e-12)


def test_measurement_rows():
    H, ang = ekf.h_rows(True)
    assert H.shape == (11, 9) and ang.tolist() == [False] * 3 + [True] * 5 + [False] * 3
    x = np.arange(9.0)
    assert np.allclose(H @ x, [0, 1, 2, 3, 4, 5, 3, 4, 6, 7, 8])
    H, ang = ekf.h_rows(False)
    assert H.shape == (9, 9) and np.allclose(H, np.eye(9))


def _static_filter(n_up=1, P0=None, dt=0.01):
    P0 = np.diag(np.linspace(0.5, 2.0, 9)) if P0 is None else P0
    e = ekf.Ekf(np.zeros(9), P0, np.zeros((9, 9)), dt=dt, n_up=n_up)
    return e


def _rest_input():
    return np.r_[0, 0, ekf.G0, 0, 0, 0]


def test_update_is_the_textbook_linear_gaussian_posterior():
    # state at rest, Q = 0, H = I: after one measurement the posterior is the information-form fusion of prior and z
    e = _static_filter()
    P0 = e.P.copy()
    R = np.diag(np.linspace(0.1, 0.9, 9))
    z = np.array([0.3, -0.2, 0.1, 0.01, -0.02, 0.03, 0.5, 0.0, -0.1])
    e.push_measurement(z, R, cycle_s=0)
    e.predict(_rest_input())
    F = ekf.jacobian_f(np.zeros(9), _rest_input(), 0.01)
    Pp = F @ P0 @ F.T
    Ppost = np.linalg.inv(np.linalg.inv(Pp) + np.linalg.inv(R))
    xpost = Ppost @ (np.linalg.inv(R) @ z)                # prior mean 0; Eq. 11 with x_s = 0 leaves z unchanged up to H(x_k - x_s) = 0
    assert np.allclose(e.P, Ppost, atol=1e-12)
    assert np.allclose(e.x, xpost, atol=1e-12)


def test_upsampled_correction_equals_single_correction_for_a_static_linear_system():
    R = np.diag(np.linspace(0.1, 0.9, 9))
    z = np.array([0.3, -0.2, 0.1, 0.0, 0.0, 0.02, 0.0, 0.0, 0.0])
    P0 = np.diag([1.0] * 3 + [1e-3] * 3 + [1e-9] * 3)     # velocity pinned to 0 so the prediction is the identity on position
    one = _static_filter(1, P0)
    one.push_measurement(z, R, 0)
    one.predict(_rest_input())
    ten = _static_filter(10, P0)
    ten.push_measurement(z, R, 0)
    for _ in range(10):
        ten.predict(_rest_input())
    assert np.allclose(ten.x[:6], one.x[:6], atol=2e-5)      # not exactly static: gravity couples attitude into velocity
    assert np.allclose(np.diag(ten.P)[:6], np.diag(one.P)[:6], rtol=1e-3)
    # and the correction really is spread: after one cycle only a fraction has been applied
    part = _static_filter(10, P0)
    part.push_measurement(z, R, 0)
    part.predict(_rest_input())
    assert 0.05 < part.x[0] / one.x[0] < 0.7          # first of ten steps: K = P/(P + 10 R) = 0.15 of z vs 0.27 in total


def test_delay_compensation_eq11_extrapolates_the_measurement_with_the_predicted_motion():
    # the vehicle drives straight at 50 m/s; a perfect position fix taken 8 cycles ago arrives now: with Eq. 11 the
    # state must stay on the true trajectory (no jump back by 8 cycles * 0.5 m)
    dt = 0.01
    x0 = np.r_[0, 0, 0, 0, 0, 0, 50.0, 0, 0]
    e = ekf.Ekf(x0, np.eye(9) * 1e-2, np.eye(9) * 1e-8, dt=dt)
    u = _rest_input()
    for _ in range(20):
        e.predict(u)
    truth_s = e.history[12].copy()
    R = np.eye(9) * 1e-6
    e.push_measurement(truth_s, R, cycle_s=12)            # z_s = h(x_s) exactly: innovation zero
    before = e.x.copy()
    e.predict(u)
    assert np.allclose(e.x, ekf.f(before, u, dt), atol=1e-9)
    # a fix that says "you were 0.2 m further left at cycle 12" moves the CURRENT state 0.2 m left, not back in time
    e2 = ekf.Ekf(x0, np.eye(9) * 1e-2, np.eye(9) * 1e-8, dt=dt)
    for _ in range(20):
        e2.predict(u)
    z = e2.history[12].copy(); z[1] += 0.2
    e2.push_measurement(z, R, cycle_s=12)
    e2.predict(u)
    assert abs(e2.x[1] - 0.2) < 2e-3 and abs(e2.x[0] - 50.0 * 21 * dt) < 2e-3


def test_angle_innovation_is_wrapped():
    x0 = np.r_[0, 0, 0, 0, 0, np.pi - 0.01, 0, 0, 0]
    e = ekf.Ekf(x0, np.eye(9) * 1e-2, np.zeros((9, 9)))
    z = x0.copy(); z[5] = -np.pi + 0.01                   # 0.02 rad away through the wrap, not 2 pi - 0.02
    e.push_measurement(z, np.eye(9) * 1e-2, 0)
    e.predict(_rest_input())
    assert abs(ekf.wrap(e.x[5] - x0[5])) < 0.02
