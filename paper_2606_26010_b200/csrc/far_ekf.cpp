// far_ekf.cpp -- HOST-only FP64 Sensor Fusion backend: the kinematic EKF of PAPER.md:113-128
// (Eq. 8-10), delay compensation and measurement up-sampling (Eq. 11) and the LiDAR velocity of
// Eq. 7.  Readings R18-R20 in DESIGN.md.  Not a kernel: it runs at 100 Hz on a few dozen doubles
// and only hands the GPU path its two inputs (initial guess, velocity history).
#include <cmath>
#include <cstdint>
#include <cstring>
#include <new>
#include <vector>

#include "../../include/far.h"

namespace {

constexpr double G0 = 9.80665;
constexpr int NX = 9;
constexpr int HIST = 512;       // cycles of state / twist history (5.12 s at 100 Hz)
constexpr int MAXZ = 11;

struct Trig { double sr, cr, sp, cp, sy, cy; };
inline Trig trig(const double* th) { return {std::sin(th[0]), std::cos(th[0]), std::sin(th[1]), std::cos(th[1]), std::sin(th[2]), std::cos(th[2])}; }

// R = Rz(yaw) Ry(pitch) Rx(roll), row-major
inline void rot_zyx(const Trig& t, double R[9]) {
    R[0] = t.cy * t.cp; R[1] = t.cy * t.sp * t.sr - t.sy * t.cr; R[2] = t.cy * t.sp * t.cr + t.sy * t.sr;
    R[3] = t.sy * t.cp; R[4] = t.sy * t.sp * t.sr + t.cy * t.cr; R[5] = t.sy * t.sp * t.cr - t.cy * t.sr;
    R[6] = -t.sp;       R[7] = t.cp * t.sr;                      R[8] = t.cp * t.cr;
}

// Eq. 9 (R18) and, if F != nullptr, its analytic Jacobian F = I + dt * d(xdot)/dx
void model(const double* x, const double* a, const double* w, double dt, double* xn, double* F) {
    const double* th = x + 3;
    const double* v = x + 6;
    const Trig t = trig(th);
    double R[9];
    rot_zyx(t, R);
    const double tp = t.sp / t.cp;
    double xd[9];
    for (int i = 0; i < 3; ++i) xd[i] = R[3 * i] * v[0] + R[3 * i + 1] * v[1] + R[3 * i + 2] * v[2];
    const double sqr = t.sr * w[1] + t.cr * w[2];     // s_phi q + c_phi r
    const double cqr = t.cr * w[1] - t.sr * w[2];     // c_phi q - s_phi r
    xd[3] = w[0] + tp * sqr;
    xd[4] = cqr;
    xd[5] = sqr / t.cp;
    // g(theta) = R^T (0, 0, -g0) = -g0 * (third row of R)
    const double gb[3] = {-G0 * R[6], -G0 * R[7], -G0 * R[8]};
    xd[6] = -(w[1] * v[2] - w[2] * v[1]) + a[0] + gb[0];
    xd[7] = -(w[2] * v[0] - w[0] * v[2]) + a[1] + gb[1];
    xd[8] = -(w[0] * v[1] - w[1] * v[0]) + a[2] + gb[2];
    for (int i = 0; i < NX; ++i) xn[i] = x[i] + dt * xd[i];
    if (!F) return;
    double J[81];
    std::memset(J, 0, sizeof(J));
    // d(R v)/d theta: columns = (dR/droll) v, (dR/dpitch) v, (dR/dyaw) v
    const double dRr[9] = {0, t.cy * t.sp * t.cr + t.sy * t.sr, -t.cy * t.sp * t.sr + t.sy * t.cr,
                           0, t.sy * t.sp * t.cr - t.cy * t.sr, -t.sy * t.sp * t.sr - t.cy * t.cr,
                           0, t.cp * t.cr, -t.cp * t.sr};
    const double dRp[9] = {-t.cy * t.sp, t.cy * t.cp * t.sr, t.cy * t.cp * t.cr,
                           -t.sy * t.sp, t.sy * t.cp * t.sr, t.sy * t.cp * t.cr,
                           -t.cp, -t.sp * t.sr, -t.sp * t.cr};
    const double dRy[9] = {-R[3], -R[4], -R[5], R[0], R[1], R[2], 0, 0, 0};
    for (int i = 0; i < 3; ++i) {
        J[9 * i + 3] = dRr[3 * i] * v[0] + dRr[3 * i + 1] * v[1] + dRr[3 * i + 2] * v[2];
        J[9 * i + 4] = dRp[3 * i] * v[0] + dRp[3 * i + 1] * v[1] + dRp[3 * i + 2] * v[2];
        J[9 * i + 5] = dRy[3 * i] * v[0] + dRy[3 * i + 1] * v[1] + dRy[3 * i + 2] * v[2];
        for (int j = 0; j < 3; ++j) J[9 * i + 6 + j] = R[3 * i + j];
    }
    // d(E w)/d theta
    const double c2 = t.cp * t.cp;
    J[9 * 3 + 3] = tp * cqr;        J[9 * 3 + 4] = sqr / c2;
    J[9 * 4 + 3] = -sqr;
    J[9 * 5 + 3] = cqr / t.cp;      J[9 * 5 + 4] = sqr * t.sp / c2;
    // d g(theta)/d theta : g = -g0 (-sp, cp sr, cp cr)
    J[9 * 6 + 4] = -G0 * (-t.cp);
    J[9 * 7 + 3] = -G0 * (t.cp * t.cr);   J[9 * 7 + 4] = -G0 * (-t.sp * t.sr);
    J[9 * 8 + 3] = -G0 * (-t.cp * t.sr);  J[9 * 8 + 4] = -G0 * (-t.sp * t.cr);
    // d(-[w]x v)/d v = -[w]x
    J[9 * 6 + 7] += w[2];  J[9 * 6 + 8] += -w[1];
    J[9 * 7 + 6] += -w[2]; J[9 * 7 + 8] += w[0];
    J[9 * 8 + 6] += w[1];  J[9 * 8 + 7] += -w[0];
    for (int i = 0; i < 81; ++i) F[i] = dt * J[i];
    for (int i = 0; i < NX; ++i) F[9 * i + i] += 1.0;
}

inline double wrap_pi(double a) {
    const double two_pi = 6.283185307179586476925286766559;
    a = std::fmod(a + 3.14159265358979323846, two_pi);
    if (a < 0) a += two_pi;
    return a - 3.14159265358979323846;
}

// (roll, pitch, yaw) of R = Rz Ry Rx
inline void euler_zyx(const double R[9], double th[3]) {
    th[1] = std::asin(std::fmax(-1.0, std::fmin(1.0, -R[6])));
    th[0] = std::atan2(R[7], R[8]);
    th[2] = std::atan2(R[3], R[0]);
}

// in-place inverse of a symmetric positive definite m x m matrix (m <= 11) by Gauss-Jordan with partial pivoting
bool invert(double* A, int m) {
    double B[MAXZ * MAXZ];
    for (int i = 0; i < m; ++i) for (int j = 0; j < m; ++j) B[i * m + j] = i == j ? 1.0 : 0.0;
    for (int c = 0; c < m; ++c) {
        int piv = c;
        for (int r = c + 1; r < m; ++r) if (std::fabs(A[r * m + c]) > std::fabs(A[piv * m + c])) piv = r;
        if (!(std::fabs(A[piv * m + c]) > 0.0)) return false;
        if (piv != c) for (int j = 0; j < m; ++j) { std::swap(A[c * m + j], A[piv * m + j]); std::swap(B[c * m + j], B[piv * m + j]); }
        const double d = 1.0 / A[c * m + c];
        for (int j = 0; j < m; ++j) { A[c * m + j] *= d; B[c * m + j] *= d; }
        for (int r = 0; r < m; ++r) {
            if (r == c) continue;
            const double f = A[r * m + c];
            if (f == 0.0) continue;
            for (int j = 0; j < m; ++j) { A[r * m + j] -= f * A[c * m + j]; B[r * m + j] -= f * B[c * m + j]; }
        }
    }
    std::memcpy(A, B, sizeof(double) * m * m);
    return true;
}

struct Pending {
    double z[MAXZ], Rd[MAXZ], xs[NX];
    int m;            // 9 or 11
    int remaining;
};

}  // namespace

struct far_ekf {
    double x[NX], P[81], Q[NX], dt, ab[3], wb[3];
    int n_up;
    int64_t k;
    double hist_x[HIST][NX];
    double hist_tw[HIST][6];
    std::vector<Pending> pending;
};

namespace {

const int ROWS9[9] = {0, 1, 2, 3, 4, 5, 6, 7, 8};
const int ROWS11[11] = {0, 1, 2, 3, 4, 5, 3, 4, 6, 7, 8};     // Eq. 10 (R19): (t, theta, theta_ref = roll/pitch, v)

// one (partial) correction with the delay-compensated measurement (Eq. 11, R20)
void correct(far_ekf* e, Pending& p) {
    const int m = p.m;
    const int* rows = m == 11 ? ROWS11 : ROWS9;
    double y[MAXZ];
    for (int i = 0; i < m; ++i) {
        // z_k = z_s + h(x_k|k-1) - h(x_s);  innovation y = z_k - h(x_k|k-1)
        const double zk = p.z[i] + e->x[rows[i]] - p.xs[rows[i]];
        y[i] = zk - e->x[rows[i]];
        if (rows[i] >= 3 && rows[i] <= 5) y[i] = wrap_pi(y[i]);
    }
    double S[MAXZ * MAXZ];
    for (int i = 0; i < m; ++i)
        for (int j = 0; j < m; ++j) S[i * m + j] = e->P[9 * rows[i] + rows[j]] + (i == j ? p.Rd[i] * e->n_up : 0.0);
    if (!invert(S, m)) return;
    double K[NX * MAXZ];                       // K = P H^T S^-1
    for (int a = 0; a < NX; ++a)
        for (int j = 0; j < m; ++j) {
            double s = 0.0;
            for (int i = 0; i < m; ++i) s += e->P[9 * a + rows[i]] * S[i * m + j];
            K[a * m + j] = s;
        }
    double dx[NX];
    for (int a = 0; a < NX; ++a) {
        double s = 0.0;
        for (int j = 0; j < m; ++j) s += K[a * m + j] * y[j];
        dx[a] = s;
        e->x[a] += s;
        p.xs[a] += s;                          // R20: what this measurement has already corrected
    }
    // Joseph form: P = (I - K H) P (I - K H)^T + K (n_up R) K^T
    double A[81], AP[81], Pn[81];
    for (int a = 0; a < NX; ++a)
        for (int b = 0; b < NX; ++b) {
            double kh = 0.0;
            for (int j = 0; j < m; ++j) if (rows[j] == b) kh += K[a * m + j];
            A[9 * a + b] = (a == b ? 1.0 : 0.0) - kh;
        }
    for (int a = 0; a < NX; ++a)
        for (int b = 0; b < NX; ++b) {
            double s = 0.0;
            for (int c = 0; c < NX; ++c) s += A[9 * a + c] * e->P[9 * c + b];
            AP[9 * a + b] = s;
        }
    for (int a = 0; a < NX; ++a)
        for (int b = 0; b < NX; ++b) {
            double s = 0.0;
            for (int c = 0; c < NX; ++c) s += AP[9 * a + c] * A[9 * b + c];
            for (int j = 0; j < m; ++j) s += K[a * m + j] * (p.Rd[j] * e->n_up) * K[b * m + j];
            Pn[9 * a + b] = s;
        }
    std::memcpy(e->P, Pn, sizeof(Pn));
}

}  // namespace

extern "C" {

far_ekf_t* far_ekf_create(const double x0[9], const double P0_diag[9], const double Q_diag[9], double dt, int32_t n_up,
                          const double accel_bias[3], const double gyro_bias[3]) {
    if (!x0 || !P0_diag || !Q_diag || !(dt > 0.0) || n_up < 1) return nullptr;
    far_ekf* e = new (std::nothrow) far_ekf();
    if (!e) return nullptr;
    std::memcpy(e->x, x0, sizeof(e->x));
    std::memset(e->P, 0, sizeof(e->P));
    for (int i = 0; i < NX; ++i) { e->P[9 * i + i] = P0_diag[i]; e->Q[i] = Q_diag[i]; }
    e->dt = dt;
    e->n_up = n_up;
    for (int i = 0; i < 3; ++i) { e->ab[i] = accel_bias ? accel_bias[i] : 0.0; e->wb[i] = gyro_bias ? gyro_bias[i] : 0.0; }
    e->k = 0;
    std::memset(e->hist_x, 0, sizeof(e->hist_x));
    std::memset(e->hist_tw, 0, sizeof(e->hist_tw));
    std::memcpy(e->hist_x[0], e->x, sizeof(e->x));
    return e;
}

void far_ekf_destroy(far_ekf_t* e) { delete e; }

int64_t far_ekf_predict(far_ekf_t* e, const double accel_m[3], const double gyro_m[3]) {
    if (!e || !accel_m || !gyro_m) return -1;
    double F[81], xn[NX], FP[81], Pn[81];
    const double a[3] = {accel_m[0] - e->ab[0], accel_m[1] - e->ab[1], accel_m[2] - e->ab[2]};
    const double w[3] = {gyro_m[0] - e->wb[0], gyro_m[1] - e->wb[1], gyro_m[2] - e->wb[2]};
    {
        // Eq. 9 prints -[w_m]x v with the measured rate and E(theta)(w_m - w_b), a_m - a_b with the corrected ones (R18).
        // The Jacobian is that of the step actually taken: its position / attitude rows with the corrected rate, its
        // velocity rows with the measured one
        double xb[NX], Fb[81];
        model(e->x, a, w, e->dt, xb, Fb);
        double xr[NX], Fr[81];
        model(e->x, a, gyro_m, e->dt, xr, Fr);
        for (int i = 0; i < 6; ++i) xn[i] = xb[i];
        for (int i = 6; i < 9; ++i) xn[i] = xr[i];
        std::memcpy(F, Fb, 6 * 9 * sizeof(double));
        std::memcpy(F + 6 * 9, Fr + 6 * 9, 3 * 9 * sizeof(double));
    }
    for (int i = 0; i < NX; ++i)
        for (int j = 0; j < NX; ++j) {
            double s = 0.0;
            for (int c = 0; c < NX; ++c) s += F[9 * i + c] * e->P[9 * c + j];
            FP[9 * i + j] = s;
        }
    for (int i = 0; i < NX; ++i)
        for (int j = 0; j < NX; ++j) {
            double s = 0.0;
            for (int c = 0; c < NX; ++c) s += FP[9 * i + c] * F[9 * j + c];
            Pn[9 * i + j] = s + (i == j ? e->Q[i] : 0.0);
        }
    std::memcpy(e->P, Pn, sizeof(Pn));
    std::memcpy(e->x, xn, sizeof(xn));
    e->k += 1;
    for (auto& p : e->pending) { correct(e, p); p.remaining -= 1; }
    size_t keep = 0;
    for (size_t i = 0; i < e->pending.size(); ++i) if (e->pending[i].remaining > 0) e->pending[keep++] = e->pending[i];
    e->pending.resize(keep);
    const int slot = (int)(e->k % HIST);
    std::memcpy(e->hist_x[slot], e->x, sizeof(e->x));
    for (int i = 0; i < 3; ++i) { e->hist_tw[slot][i] = e->x[6 + i]; e->hist_tw[slot][3 + i] = w[i]; }
    return e->k;
}

int far_ekf_push_lidar(far_ekf_t* e, const far_pose_t* T_L, const double v_L[3], const double theta_ref[2],
                       const double R_diag[], int64_t cycle_s) {
    if (!e || !T_L || !v_L || !R_diag) return FAR_ERR_ARG;
    if (cycle_s < 0 || cycle_s > e->k || e->k - cycle_s >= HIST) return FAR_ERR_ARG;
    Pending p;
    p.m = theta_ref ? 11 : 9;
    double th[3];
    euler_zyx(T_L->R, th);
    int q = 0;
    for (int i = 0; i < 3; ++i) p.z[q++] = T_L->t[i];
    for (int i = 0; i < 3; ++i) p.z[q++] = th[i];
    if (theta_ref) { p.z[q++] = theta_ref[0]; p.z[q++] = theta_ref[1]; }
    for (int i = 0; i < 3; ++i) p.z[q++] = v_L[i];
    for (int i = 0; i < p.m; ++i) {
        if (!(R_diag[i] > 0.0)) return FAR_ERR_ARG;
        p.Rd[i] = R_diag[i];
    }
    std::memcpy(p.xs, e->hist_x[cycle_s % HIST], sizeof(p.xs));
    p.remaining = e->n_up;
    e->pending.push_back(p);
    return FAR_OK;
}

int far_ekf_state(const far_ekf_t* e, double x[9], double* P, int64_t* cycle) {
    if (!e || !x) return FAR_ERR_ARG;
    std::memcpy(x, e->x, sizeof(e->x));
    if (P) std::memcpy(P, e->P, sizeof(e->P));
    if (cycle) *cycle = e->k;
    return FAR_OK;
}

int far_ekf_pose(const far_ekf_t* e, far_pose_t* out) {
    if (!e || !out) return FAR_ERR_ARG;
    rot_zyx(trig(e->x + 3), out->R);
    for (int i = 0; i < 3; ++i) out->t[i] = e->x[i];
    return FAR_OK;
}

int far_ekf_velocity_history(const far_ekf_t* e, int32_t m, double* times, double* vel6) {
    if (!e || m < 1 || !times || !vel6) return 0;
    int64_t n = e->k < m ? e->k : m;
    if (n > HIST - 1) n = HIST - 1;
    for (int64_t j = 0; j < n; ++j) {
        const int64_t c = e->k - n + 1 + j;
        times[j] = (double)c * e->dt;
        std::memcpy(vel6 + 6 * j, e->hist_tw[c % HIST], 6 * sizeof(double));
    }
    return (int)n;
}

int far_lidar_velocity(const far_pose_t* T_t, const far_pose_t* T_prev, double dt, double v_out[3]) {
    if (!T_t || !T_prev || !v_out || !(dt > 0.0)) return FAR_ERR_ARG;
    const double d[3] = {T_t->t[0] - T_prev->t[0], T_t->t[1] - T_prev->t[1], T_t->t[2] - T_prev->t[2]};
    for (int i = 0; i < 3; ++i) v_out[i] = (T_t->R[i] * d[0] + T_t->R[3 + i] * d[1] + T_t->R[6 + i] * d[2]) / dt;   // R^T d / dt
    return FAR_OK;
}

int far_ekf_model(const double x[9], const double u[6], double dt, double x_next[9], double F[81]) {
    if (!x || !u || !x_next) return FAR_ERR_ARG;
    model(x, u, u + 3, dt, x_next, F);
    return FAR_OK;
}

}  // extern "C"
