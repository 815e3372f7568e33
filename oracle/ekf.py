"""ORACLE (test infrastructure, not the product): the kinematic EKF of the Sensor Fusion module, SURVEY 8(f)-3.

Plain NumPy FP64 restatement of PAPER.md:113-136 (Eq. 8-11) and Eq. 7, step by step in the paper's
order and notation.  Shares no code with paper_2606_26010_b200/; only tests/ may import it.  Readings R18-R20:

R18  Eq. 9 prints x_{k-1} + [...] without a step: the bracket is the state derivative and is multiplied by dt (explicit
     Euler, dt = 1/100 s at the paper's 100 Hz).  theta = (roll, pitch, yaw), R(theta) = Rz(yaw) Ry(pitch) Rx(roll) maps
     body to map, E(theta) maps body rates to Euler-angle rates, g(theta) = R(theta)^T (0, 0, -g0) is gravity seen in the
     body frame (the accelerometer measures specific force, so a = a_m - a_b + g(theta)); -[w_m]x v is the transport term
     of a velocity expressed in the rotating body frame.  The Jacobian F = d f / d x is taken by central differences here
     (the product uses the analytic one: the two are compared in the tests).
R19  Eq. 10: z = (t_L, theta_L, theta_ref, v_L) in R^11 with theta_ref = reference (roll, pitch); h(x) is linear, a row
     selection of x: [t; theta; theta[0:2]; v].  The paper does not give the formulas of theta_ref ([31],[32]): the
     reference angles are an INPUT here (rows are dropped when none is given, z in R^9).  Angle residuals are wrapped
     to (-pi, pi].
R20  Eq. 11 z_k = z_s + h(x_k|k-1) - h(x_s) with x_s the stored state at the measurement's time stamp (nearest stored
     cycle).  "upsample the measurements and distribute their influence ... over multiple update cycles": a measurement
     is applied in n_up consecutive cycles, each time re-extrapolated by Eq. 11 and with its covariance multiplied by
     n_up; the reference state x_s of that measurement is moved by every correction the measurement has already
     applied (so a partial step sees the innovation that is still left).  For a linear static system the n_up partial
     corrections then equal the single full one exactly (sequential fusion of n_up measurements of covariance n_up R).
"""
from __future__ import annotations

import numpy as np

G0 = 9.80665


def rot(theta):
    """R(theta) = Rz(yaw) Ry(pitch) Rx(roll): body -> map"""
    r, p, y = theta
    cr, sr, cp, sp, cy, sy = np.cos(r), np.sin(r), np.cos(p), np.sin(p), np.cos(y), np.sin(y)
    Rx = np.array([[1, 0, 0], [0, cr, -sr], [0, sr, cr]])
    Ry = np.array([[cp, 0, sp], [0, 1, 0], [-sp, 0, cp]])
    Rz = np.array([[cy, -sy, 0], [sy, cy, 0], [0, 0, 1]])
    return Rz @ Ry @ Rx


def euler_rates(theta):
    """E(theta): body angular velocity -> (roll, pitch, yaw) rates for the ZYX convention"""
    r, p, _ = theta
    cr, sr, cp, tp = np.cos(r), np.sin(r), np.cos(p), np.tan(p)
    return np.array([[1, sr * tp, cr * tp], [0, cr, -sr], [0, sr / cp, cr / cp]])


def hat(w):
    return np.array([[0, -w[2], w[1]], [w[2], 0, -w[0]], [-w[1], w[0], 0]])


def f(x, u, dt, a_b=np.zeros(3), w_b=np.zeros(3)):
    """Eq. 9 (R18): x = (t, theta, v), u = (a_m, w_m)"""
    x = np.asarray(x, dtype=np.float64)
    t, th, v = x[0:3], x[3:6], x[6:9]
    a_m, w_m = np.asarray(u[0:3], dtype=np.float64), np.asarray(u[3:6], dtype=np.float64)
    g_body = rot(th).T @ np.array([0.0, 0.0, -G0])
    dx = np.concatenate([rot(th) @ v,
                         euler_rates(th) @ (w_m - w_b),
                         -hat(w_m) @ v + (a_m - a_b) + g_body])
    return x + dx * dt


def jacobian_f(x, u, dt, a_b=None, w_b=None, eps=1e-6):
    """F = d f / d x of the step ACTUALLY taken (Eq. 9 with the bias-corrected inputs where it uses them), by central
    differences"""
    kw = {} if a_b is None and w_b is None else dict(a_b=a_b, w_b=w_b)
    F = np.zeros((9, 9))
    for j in range(9):
        d = np.zeros(9)
        d[j] = eps
        F[:, j] = (f(x + d, u, dt, **kw) - f(x - d, u, dt, **kw)) / (2 * eps)
    return F


def h_rows(with_ref):
    """Eq. 10 (R19): row selection of the 9-state for z = (t_L, theta_L, [theta_ref], v_L)"""
    rows = [0, 1, 2, 3, 4, 5] + ([3, 4] if with_ref else []) + [6, 7, 8]
    H = np.zeros((len(rows), 9))
    for i, r in enumerate(rows):
        H[i, r] = 1.0
    angle = np.array([3 <= r <= 5 for r in rows])
    return H, angle


def wrap(a):
    return (a + np.pi) % (2 * np.pi) - np.pi


def lidar_velocity(R_t, t_t, t_prev, dt):
    """Eq. 7: v_L = R_L,t^-1 (t_t - t_{t-1}) / dt"""
    return np.asarray(R_t).T @ (np.asarray(t_t) - np.asarray(t_prev)) / dt


class Ekf:
    def __init__(self, x0, P0, Q, dt=0.01, n_up=1, a_b=np.zeros(3), w_b=np.zeros(3)):
        self.x = np.asarray(x0, dtype=np.float64).copy()
        self.P = np.asarray(P0, dtype=np.float64).copy()
        self.Q = np.asarray(Q, dtype=np.float64).copy()
        self.dt, self.n_up = float(dt), int(n_up)
        self.a_b, self.w_b = np.asarray(a_b, float), np.asarray(w_b, float)
        self.k = 0
        self.history = {0: self.x.copy()}            # cycle index -> state after that cycle (the EKF's state history)
        self.pending = []                             # [z_s, R, with_ref, x_s, remaining]

    def predict(self, u):
        """one 100 Hz cycle: x_k|k-1 = f(x_k-1, u_k), P = F P F^T + Q; then the pending (up-sampled) corrections"""
        F = jacobian_f(self.x, u, self.dt, self.a_b, self.w_b)
        self.x = f(self.x, u, self.dt, self.a_b, self.w_b)
        self.P = F @ self.P @ F.T + self.Q
        self.k += 1
        for m in self.pending:
            self._correct(m)
            m[4] -= 1
        self.pending = [m for m in self.pending if m[4] > 0]
        self.history[self.k] = self.x.copy()
        return self.x

    def push_measurement(self, z_s, R, cycle_s, with_ref=False):
        """a LiDAR measurement taken at cycle `cycle_s` (<= current cycle), arriving now: queued for n_up cycles"""
        x_s = self.history[int(cycle_s)]
        self.pending.append([np.asarray(z_s, float), np.asarray(R, float), bool(with_ref), x_s.copy(), self.n_up])

    def _correct(self, m):
        z_s, R, with_ref, x_s, _ = m
        H, angle = h_rows(with_ref)
        z_k = z_s + H @ self.x - H @ x_s                 # Eq. 11
        y = z_k - H @ self.x
        y[angle] = wrap(y[angle])
        S = H @ self.P @ H.T + R * self.n_up             # R20: covariance inflated by n_up
        K = self.P @ H.T @ np.linalg.inv(S)
        dx = K @ y
        self.x = self.x + dx
        m[3] = x_s + dx                                  # R20: what this measurement has already corrected
        I_KH = np.eye(9) - K @ H
        self.P = I_KH @ self.P @ I_KH.T + K @ (R * self.n_up) @ K.T     # Joseph form
