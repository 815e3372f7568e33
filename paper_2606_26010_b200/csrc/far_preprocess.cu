// far_preprocess.cu -- motion undistortion of a LiDAR sweep.
//
// PAPER.md:56 "the distortion of the LiDAR scan is corrected using the velocity history of the Sensor Fusion.  We
// perform a linear regression on both the linear and angular velocities to efficiently model the LiDAR's motion
// during scanning.  This continuous motion model is evaluated in CUDA, effectively processing all points in
// parallel.  Consequently, each raw point is undistorted and projected to the frame reference timestamp, which is
// equal to the scan's final point-timestamp."  Readings R15 (least-squares twist line) and R16 (Magnus expansion
// of that line to second order, SE(3) exponential of R12) in DESIGN.md.
//
// B200 design: one pass, one thread per point (grid-stride), nothing but the point, its time offset and the result
// crosses HBM (16 B in, 12 B out at stride 3).  The twelve line coefficients and the bracket [a,b]/12 are kernel
// arguments (constant bank).  All arithmetic is FP64 -- the result is rounded to fp32 once -- and the rotation is
// applied as p + A (phi x p) + B (phi x (phi x p)) without ever forming a matrix; for the small angles of a sweep
// (|phi| <= 0.5 rad) the coefficients A = sin(t)/t, B = (1-cos t)/t^2, C = (t-sin t)/t^3 come from their Taylor
// series in t^2 (5 terms up to 0.1 rad, 9 terms up to 0.5 rad; remainders < 3e-18), which avoids sincos, the square root
// and two divisions.
#include <cmath>
#include <cstdlib>
#include <cstring>

#include "far_internal.h"

using namespace far;

namespace far {

struct MotionArgs {
    double a[6], b[6], c[6];   // xi(t) = a + b (t - t_ref);  c = [a, b] / 12
    double dt_ref;
};

__device__ __forceinline__ void abc_coefficients(double x /* theta^2 */, double& A, double& B, double& C) {
    if (x <= 0.01) {
        // |phi| <= 0.1 rad (every realistic sweep: 1 rad/s over 0.1 s): 5 terms, remainder x^5 / 11! < 3e-18
        A = 1.0 / 362880.0;                      B = 1.0 / 3628800.0;                     C = 1.0 / 39916800.0;
        A = fma(A, x, -1.0 / 5040.0);            B = fma(B, x, -1.0 / 40320.0);           C = fma(C, x, -1.0 / 362880.0);
        A = fma(A, x, 1.0 / 120.0);              B = fma(B, x, 1.0 / 720.0);              C = fma(C, x, 1.0 / 5040.0);
        A = fma(A, x, -1.0 / 6.0);               B = fma(B, x, -1.0 / 24.0);              C = fma(C, x, -1.0 / 120.0);
        A = fma(A, x, 1.0);                      B = fma(B, x, 0.5);                      C = fma(C, x, 1.0 / 6.0);
    } else if (x <= 0.25) {
        // sum_k (-1)^k x^k / (2k+1)!, / (2k+2)!, / (2k+3)!   for k = 0..8 (Horner)
        A = -1.0 / 355687428096000.0;      // 17!
        B = -1.0 / 6402373705728000.0;     // 18!
        C = -1.0 / 121645100408832000.0;   // 19!
        A = fma(A, x, 1.0 / 1307674368000.0);   B = fma(B, x, 1.0 / 20922789888000.0);   C = fma(C, x, 1.0 / 355687428096000.0);
        A = fma(A, x, -1.0 / 6227020800.0);     B = fma(B, x, -1.0 / 87178291200.0);     C = fma(C, x, -1.0 / 1307674368000.0);
        A = fma(A, x, 1.0 / 39916800.0);        B = fma(B, x, 1.0 / 479001600.0);        C = fma(C, x, 1.0 / 6227020800.0);
        A = fma(A, x, -1.0 / 362880.0);         B = fma(B, x, -1.0 / 3628800.0);         C = fma(C, x, -1.0 / 39916800.0);
        A = fma(A, x, 1.0 / 5040.0);            B = fma(B, x, 1.0 / 40320.0);            C = fma(C, x, 1.0 / 362880.0);
        A = fma(A, x, -1.0 / 120.0);            B = fma(B, x, -1.0 / 720.0);             C = fma(C, x, -1.0 / 5040.0);
        A = fma(A, x, 1.0 / 6.0);               B = fma(B, x, 1.0 / 24.0);               C = fma(C, x, 1.0 / 120.0);
        A = fma(A, -x, 1.0);                    B = fma(B, -x, 0.5);                     C = fma(C, -x, 1.0 / 6.0);
    } else {
        const double th = sqrt(x);
        double sn, cs;
        sincos(th, &sn, &cs);
        A = sn / th;
        B = (1.0 - cs) / x;
        C = (th - sn) / (x * th);
    }
}

__device__ __forceinline__ void undistort_point(const MotionArgs& M, float sx, float sy, float sz, float tm, float out[3]) {
    if (!(isfinite(sx) && isfinite(sy) && isfinite(sz) && isfinite(tm))) { out[0] = sx; out[1] = sy; out[2] = sz; return; }
    const double D = M.dt_ref - (double)tm;
    const double h = 0.5 * (D * D);
    const double g = (D * D) * D;          // c already holds the 1/12
    double o[6];                           // -(Omega_1 + Omega_2)
#pragma unroll
    for (int c = 0; c < 6; ++c) o[c] = -((M.a[c] * D - M.b[c] * h) + M.c[c] * g);
    const double rx = o[0], ry = o[1], rz = o[2], fx = o[3], fy = o[4], fz = o[5];
    double A, B, C;
    abc_coefficients(fx * fx + fy * fy + fz * fz, A, B, C);
    const double px = (double)sx, py = (double)sy, pz = (double)sz;
    // R p = p + A (phi x p) + B (phi x (phi x p));  V rho = rho + B (phi x rho) + C (phi x (phi x rho))
    const double c1x = fy * pz - fz * py, c1y = fz * px - fx * pz, c1z = fx * py - fy * px;
    const double c2x = fy * c1z - fz * c1y, c2y = fz * c1x - fx * c1z, c2z = fx * c1y - fy * c1x;
    const double d1x = fy * rz - fz * ry, d1y = fz * rx - fx * rz, d1z = fx * ry - fy * rx;
    const double d2x = fy * d1z - fz * d1y, d2y = fz * d1x - fx * d1z, d2z = fx * d1y - fy * d1x;
    out[0] = (float)((px + A * c1x + B * c2x) + (rx + B * d1x + C * d2x));
    out[1] = (float)((py + A * c1y + B * c2y) + (ry + B * d1y + C * d2y));
    out[2] = (float)((pz + A * c1z + B * c2z) + (rz + B * d1z + C * d2z));
}

// Every thread reads its point with three 4-byte loads (a warp covers 384 contiguous bytes per round of three
// instructions, so every fetched sector is fully used through L1) and writes it the same way.  A version that staged
// 1,024-point tiles through shared memory as float4 words was 27 % slower (74 vs 101 G points/s at 8 M points): the
// three block barriers per tile cost more than the vector accesses saved, the kernel being FP64-issue-bound.
__global__ void __launch_bounds__(256) undistort_kernel(const float* __restrict__ xyz, const float* __restrict__ tm,
                                                                int64_t n, int stride, MotionArgs M, float* __restrict__ out) {
    const int64_t T = (int64_t)gridDim.x * blockDim.x;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += T) {
        const float* s = xyz + i * stride;
        float o[3];
        undistort_point(M, __ldg(s), __ldg(s + 1), __ldg(s + 2), __ldg(tm + i), o);
        float* d = out + 3 * i;
        d[0] = o[0]; d[1] = o[1]; d[2] = o[2];
    }
}

}  // namespace far

extern "C" {

// R15: ordinary least squares line x(t) = a + b (t - t_ref) per twist component (host, FP64)
int far_motion_fit(const double* times, const double* vel6, int32_t m, double t_ref, far_motion_t* out) {
    if (!times || !vel6 || !out || m < 1) return FAR_ERR_ARG;
    double mean_s = 0.0;
    for (int32_t j = 0; j < m; ++j) mean_s += times[j] - t_ref;
    mean_s /= (double)m;
    double var_s = 0.0;
    for (int32_t j = 0; j < m; ++j) { const double e = (times[j] - t_ref) - mean_s; var_s += e * e; }
    for (int c = 0; c < 6; ++c) {
        double mean_x = 0.0;
        for (int32_t j = 0; j < m; ++j) mean_x += vel6[6 * j + c];
        mean_x /= (double)m;
        double cov = 0.0;
        for (int32_t j = 0; j < m; ++j) cov += ((times[j] - t_ref) - mean_s) * (vel6[6 * j + c] - mean_x);
        out->b[c] = var_s > 0.0 ? cov / var_s : 0.0;
        out->a[c] = mean_x - out->b[c] * mean_s;
    }
    return FAR_OK;
}

int far_undistort(const float* d_xyz, const float* d_time, int64_t n, int stride, double dt_ref, const far_motion_t* motion,
                  float* d_out_xyz, void* stream) {
    if (n < 0 || (stride != 3 && stride != 4) || !motion || (n > 0 && (!d_xyz || !d_time || !d_out_xyz))) return FAR_ERR_ARG;
    if (n == 0) return FAR_OK;
    MotionArgs M;
    memcpy(M.a, motion->a, sizeof(M.a));
    memcpy(M.b, motion->b, sizeof(M.b));
    const double *va = M.a, *wa = M.a + 3, *vb = M.b, *wb = M.b + 3;
    // se(3) bracket [(va,wa),(vb,wb)] = (wa x vb - wb x va, wa x wb), scaled by 1/12 (second Magnus term)
    M.c[0] = ((wa[1] * vb[2] - wa[2] * vb[1]) - (wb[1] * va[2] - wb[2] * va[1])) / 12.0;
    M.c[1] = ((wa[2] * vb[0] - wa[0] * vb[2]) - (wb[2] * va[0] - wb[0] * va[2])) / 12.0;
    M.c[2] = ((wa[0] * vb[1] - wa[1] * vb[0]) - (wb[0] * va[1] - wb[1] * va[0])) / 12.0;
    M.c[3] = (wa[1] * wb[2] - wa[2] * wb[1]) / 12.0;
    M.c[4] = (wa[2] * wb[0] - wa[0] * wb[2]) / 12.0;
    M.c[5] = (wa[0] * wb[1] - wa[1] * wb[0]) / 12.0;
    M.dt_ref = dt_ref;
    static int sms = 0;                       // SM count of the first device used (grid sizing only)
    if (sms == 0) {
        int dev = 0, v = 148;
        FAR_CUDA(cudaGetDevice(&dev));
        FAR_CUDA(cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev));
        sms = v;
    }
    int64_t g = (n + 255) / 256;
    if (g > (int64_t)sms * 32) g = (int64_t)sms * 32;
    FAR_LAUNCH(undistort_kernel, (int)g, 256, 0, (cudaStream_t)stream, d_xyz, d_time, n, stride, M, d_out_xyz);
    FAR_CUDA(cudaGetLastError());
    return FAR_OK;
}

}  // extern "C"
