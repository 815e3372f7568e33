// far_gicp.cu -- sparsity-aware GICP registration on the voxel hashmap (A8-A10), one cooperative kernel.
//
// P0* = T_t P* (Eq. 2); per iteration: kNN-search (k = 1) of every transformed source point
// in the submap, adaptive-threshold rejection, residual d = r - T s (Eq. 3), robust least squares
// on d^T (Sigma_r + T Sigma_s T^T)^-1 d (Eq. 4) with the Cauchy kernel (Eq. 5), sparsity-aware fallback
// Sigma_r = I, Sigma_s = 0 when a covariance is missing, point update (Eq. 6) and the stop test
// ||T_L,j|| <= 5e-3.  Readings R9-R14 fix what the paper leaves open: IRLS weight on
// e = sqrt(d^T M d); left perturbation T <- Exp(delta) T with delta = (rho, phi); J = [-I | [p]x]; the pose is
// accumulated in FP64 and always applied to the ORIGINAL scan; stop on ||delta||_2; max_iters replaces the
// wall-clock limit.
//
// B200 design: a registration is a few thousand source points, i.e. latency- and issue-bound, never bandwidth-
// bound, so the whole Gauss-Newton loop is ONE persistent cooperative kernel and every iteration is organised to
// keep both the instruction count and the serial chain short:
//   phase A0 8 lanes of warp 0 transform the block's 8 source points (FP64) and take their voxel indices: one
//            instruction stream instead of 8 redundant warps; a warp's source point, covariance and flag stay in
//            registers across iterations (one memory level less per iteration);
//   phase A  one warp per source point: 27-voxel probe, bounded candidate sweep (far_common.cuh::warp_nearest), gate,
//            fetch of Sigma_r -> one correspondence record in shared memory;
//   phase B  the block's 8 correspondences are linearised by 8 lanes of warp 0 at once (the ~300 FP64 operations of
//            M, weight, J^T M J are one instruction stream for 8 points instead of 8 streams with one active lane);
//   reduce   the 29 unique terms of (H, b, chi2, n) go block -> group of 32 blocks -> grid as TAGGED rows: every
//            value travels as {lo, tag, hi, tag} (two self-validating 8-byte words, tag = launch sequence and
//            iteration), so a consumer just polls the rows it needs -- no fence, no ticket atomics -- and sums
//            them in a fixed order (deterministic, no floating-point atomics);
//   solve    block 0 / thread 0: 6x6 Cholesky, SE(3) exponential, pose update and stop test in FP64, published as
//            13 tagged words; one lane per block polls the `done` word with a short back-off, then twelve lanes fetch
//            the pose: one L2 round trip from "solved" to "next iteration" without the waiters crowding that slice.
// Measured per iteration at C2 (5,352 points, debug-only globaltimer probes): A0+A 6.8 us, B 2.1, reduce 1.8, solve 2.2,
// publish 1.1-2.0.  The arithmetic of B and solve is left exactly as it is: the C3 chain (tests/test_gpu_full_size.py)
// amplifies a 1e-16 change of one increment to 2 fp32 ulps of a stored coordinate within 12 frames, along the
// unobservable direction of the corridor.
// The host is not involved until it reads the result.
#include <cstring>

#include "far_internal.h"

using namespace far;

namespace far {

constexpr int GWARPS = 8;        // warps per block = correspondences linearised together in phase B
constexpr int NTERMS = 29;       // 21 (H upper triangle) + 6 (b) + chi2 + inlier count
constexpr int TSTRIDE = 32;      // padded row

constexpr int GROUP = 32;        // blocks per first-level reduction group
constexpr int MAX_GROUPS = 64;
constexpr int GICP_BLOCKS_PER_SM = 5;
constexpr int NPUB = 13;         // published words: R[9], t[3], done
constexpr int MAX_ITERS_LIMIT = 1000;   // the iteration index shares the 32-bit tag with the launch sequence

// device scratch of one map: [max_grid] block rows, [MAX_GROUPS] group rows, the published pose
struct GicpScratch {
    uint4* rows;      // [max_grid][TSTRIDE]
    uint4* grows;     // [MAX_GROUPS][TSTRIDE]
    uint4* pub;       // [16]: 13 published words; pub[15].x = launch sequence of this map (device-resident)
};

// one transformed source point, written by one lane of warp 0 in phase A0, read by its warp in phase A
struct Src {
    float p[3];       // T s (Eq. 2)
    int k[3];         // its voxel index
    int ok;           // 0: no point / non-finite / outside the key range
};

// one correspondence, written by its warp in phase A, read by one lane of warp 0 in phase B
struct Corr {
    float p[3];       // transformed source point
    float r[3];       // its nearest map point
    float cs[6];      // Sigma_s
    float cr[6];      // Sigma_r
    int flags;        // bit 0: correspondence accepted, bit 1: both covariances valid
};


struct GicpParams {
    const float* scan;
    const float* cov6;          // nullable
    const uint8_t* valid;       // nullable
    int64_t n;
    const int64_t* d_n;         // nullable: n = min(n, *d_n)
    int stride;
    Pose init;                  // used when d_init == nullptr
    const Pose* d_init;
    double tau2, kappa, conv_eps;
    int kernel, max_iters, linearize_only;
    GicpScratch scratch;
    far_gicp_result_t* out;
};

__device__ __forceinline__ void put_tagged(uint4* dst, double v, uint32_t tag) {
    const unsigned long long b = (unsigned long long)__double_as_longlong(v);
    asm volatile("st.relaxed.gpu.global.v4.u32 [%0], {%1, %2, %3, %4};" ::"l"(dst), "r"((uint32_t)b), "r"(tag),
                 "r"((uint32_t)(b >> 32)), "r"(tag)
                 : "memory");
}

__device__ __forceinline__ uint4 load_tagged(const uint4* src) {
    uint4 w;
    asm volatile("ld.relaxed.gpu.global.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(w.x), "=r"(w.y), "=r"(w.z), "=r"(w.w) : "l"(src) : "memory");
    return w;
}

// spins until both halves carry `tag` (volatile asm: the compiler must neither hoist the load nor assume the loop ends)
__device__ __forceinline__ double wait_tagged(const uint4* src, uint32_t tag) {
    uint4 w = load_tagged(src);
    while (w.y != tag || w.w != tag) w = load_tagged(src);
    return __longlong_as_double((long long)(((unsigned long long)w.z << 32) | w.x));
}

__device__ __forceinline__ double robust_weight(int kernel, double e2, double kappa) {
    if (kernel == FAR_KERNEL_CAUCHY) return 1.0 / (1.0 + e2 / (kappa * kappa));          // Eq. 5 as IRLS weight (R9)
    if (kernel == FAR_KERNEL_GEMAN_MCCLURE) { const double s = kappa + e2; return (kappa * kappa) / (s * s); }
    return 1.0;
}

// symmetric 3x3 inverse from the 6 unique entries (xx,xy,xz,yy,yz,zz); false if singular
__device__ __forceinline__ bool inv_sym3(const double a[6], double o[6]) {
    const double c00 = a[3] * a[5] - a[4] * a[4];
    const double c01 = a[4] * a[2] - a[1] * a[5];
    const double c02 = a[1] * a[4] - a[3] * a[2];
    const double det = a[0] * c00 + a[1] * c01 + a[2] * c02;
    if (!(det != 0.0) || !isfinite(det)) return false;
    const double id = 1.0 / det;
    o[0] = c00 * id; o[1] = c01 * id; o[2] = c02 * id;
    o[3] = (a[0] * a[5] - a[2] * a[2]) * id;
    o[4] = (a[2] * a[1] - a[0] * a[4]) * id;
    o[5] = (a[0] * a[3] - a[1] * a[1]) * id;
    return true;
}

// A9 for one correspondence: the 29 terms, written by lane 0 into s_terms
__device__ __forceinline__ void correspondence_terms(const Pose& T, const double p[3], const double r[3], bool full,
                                                      const float* cs, const float* cr, int kernel, double kappa,
                                                      double* terms) {
    const double d0 = r[0] - p[0], d1 = r[1] - p[1], d2 = r[2] - p[2];   // Eq. 3
    double M[6] = {1.0, 0.0, 0.0, 1.0, 0.0, 1.0};                        // SA fallback: Sigma_r = I, Sigma_s = 0
    if (full) {
        // S = Sigma_r + R Sigma_s R^T   (Eq. 4)
        const double s[6] = {cs[0], cs[1], cs[2], cs[3], cs[4], cs[5]};
        double RS[9];
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            const double a = T.R[3 * i], b = T.R[3 * i + 1], c = T.R[3 * i + 2];
            RS[3 * i + 0] = a * s[0] + b * s[1] + c * s[2];
            RS[3 * i + 1] = a * s[1] + b * s[3] + c * s[4];
            RS[3 * i + 2] = a * s[2] + b * s[4] + c * s[5];
        }
        double S[6];
        S[0] = (double)cr[0] + (RS[0] * T.R[0] + RS[1] * T.R[1] + RS[2] * T.R[2]);
        S[1] = (double)cr[1] + (RS[0] * T.R[3] + RS[1] * T.R[4] + RS[2] * T.R[5]);
        S[2] = (double)cr[2] + (RS[0] * T.R[6] + RS[1] * T.R[7] + RS[2] * T.R[8]);
        S[3] = (double)cr[3] + (RS[3] * T.R[3] + RS[4] * T.R[4] + RS[5] * T.R[5]);
        S[4] = (double)cr[4] + (RS[3] * T.R[6] + RS[4] * T.R[7] + RS[5] * T.R[8]);
        S[5] = (double)cr[5] + (RS[6] * T.R[6] + RS[7] * T.R[7] + RS[8] * T.R[8]);
        double Mi[6];
        if (inv_sym3(S, Mi)) {
#pragma unroll
            for (int a = 0; a < 6; ++a) M[a] = Mi[a];
        }
    }
    const double Md0 = M[0] * d0 + M[1] * d1 + M[2] * d2;
    const double Md1 = M[1] * d0 + M[3] * d1 + M[4] * d2;
    const double Md2 = M[2] * d0 + M[4] * d1 + M[5] * d2;
    const double e2 = d0 * Md0 + d1 * Md1 + d2 * Md2;
    const double w = robust_weight(kernel, e2, kappa);
    const double px = p[0], py = p[1], pz = p[2];
    // X = M A with A = [p]x :  column 0 = M(:,1) pz - M(:,2) py, column 1 = -M(:,0) pz + M(:,2) px, column 2 = M(:,0) py - M(:,1) px
    const double Mr[3][3] = {{M[0], M[1], M[2]}, {M[1], M[3], M[4]}, {M[2], M[4], M[5]}};
    double X[3][3];
#pragma unroll
    for (int r_ = 0; r_ < 3; ++r_) {
        X[r_][0] = Mr[r_][1] * pz - Mr[r_][2] * py;
        X[r_][1] = Mr[r_][2] * px - Mr[r_][0] * pz;
        X[r_][2] = Mr[r_][0] * py - Mr[r_][1] * px;
    }
    // Y = A^T X (symmetric):  row 0 = pz X[1] - py X[2], row 1 = px X[2] - pz X[0], row 2 = py X[0] - px X[1]
    const double Y00 = pz * X[1][0] - py * X[2][0], Y01 = pz * X[1][1] - py * X[2][1], Y02 = pz * X[1][2] - py * X[2][2];
    const double Y11 = px * X[2][1] - pz * X[0][1], Y12 = px * X[2][2] - pz * X[0][2];
    const double Y22 = py * X[0][2] - px * X[1][2];
    // H = w J^T M J with J = [-I | A]:  [[M, -X], [-X^T, Y]];   b = w J^T M d = w [-Md ; A^T Md]
    terms[0] = w * M[0];  terms[1] = w * M[1];  terms[2] = w * M[2];  terms[3] = -w * X[0][0]; terms[4] = -w * X[0][1]; terms[5] = -w * X[0][2];
    terms[6] = w * M[3];  terms[7] = w * M[4];  terms[8] = -w * X[1][0]; terms[9] = -w * X[1][1]; terms[10] = -w * X[1][2];
    terms[11] = w * M[5]; terms[12] = -w * X[2][0]; terms[13] = -w * X[2][1]; terms[14] = -w * X[2][2];
    terms[15] = w * Y00;  terms[16] = w * Y01;  terms[17] = w * Y02;
    terms[18] = w * Y11;  terms[19] = w * Y12;
    terms[20] = w * Y22;
    terms[21] = -w * Md0; terms[22] = -w * Md1; terms[23] = -w * Md2;
    terms[24] = w * (pz * Md1 - py * Md2);
    terms[25] = w * (px * Md2 - pz * Md0);
    terms[26] = w * (py * Md0 - px * Md1);
    terms[27] = w * e2;
    terms[28] = 1.0;
}

// 6x6 Cholesky solve H x = rhs (FP64), fully unrolled so L lives in registers; one rsqrt per pivot and
// multiplications by the reciprocal pivots instead of 27 divisions (this thread is the serial section of every
// Gauss-Newton iteration).  false if H is not positive definite.
__device__ __forceinline__ bool chol_solve6(const double* H, const double* rhs, double* x) {
    double L[6][6], inv[6];
#pragma unroll
    for (int j = 0; j < 6; ++j) {
        double s = H[6 * j + j];
#pragma unroll
        for (int k = 0; k < j; ++k) s -= L[j][k] * L[j][k];
        if (!(s > 0.0) || !isfinite(s)) return false;
        inv[j] = rsqrt(s);
        L[j][j] = s * inv[j];
#pragma unroll
        for (int i = j + 1; i < 6; ++i) {
            double t = H[6 * i + j];
#pragma unroll
            for (int k = 0; k < j; ++k) t -= L[i][k] * L[j][k];
            L[i][j] = t * inv[j];
        }
    }
    double y[6];
#pragma unroll
    for (int i = 0; i < 6; ++i) {
        double t = rhs[i];
#pragma unroll
        for (int k = 0; k < i; ++k) t -= L[i][k] * y[k];
        y[i] = t * inv[i];
    }
#pragma unroll
    for (int i = 5; i >= 0; --i) {
        double t = y[i];
#pragma unroll
        for (int k = i + 1; k < 6; ++k) t -= L[k][i] * x[k];
        x[i] = t * inv[i];
    }
    return true;
}

// SE(3) exponential of delta = (rho, phi), translation first (R12); series below theta = 1e-8
__device__ __forceinline__ void se3_exp(const double* d, Pose& E) {
    const double px = d[3], py = d[4], pz = d[5];
    const double th2 = px * px + py * py + pz * pz;
    const double th = sqrt(th2);
    double A, B, C;
    if (th < 1e-8) {
        A = 1.0 - th2 / 6.0; B = 0.5 - th2 / 24.0; C = 1.0 / 6.0 - th2 / 120.0;
    } else {
        double sn, cs;
        sincos(th, &sn, &cs);
        const double ith = 1.0 / th, ith2 = ith * ith;
        A = sn * ith; B = (1.0 - cs) * ith2; C = (th - sn) * ith2 * ith;
    }
    const double K[9] = {0, -pz, py, pz, 0, -px, -py, px, 0};
    // K^2 = phi phi^T - |phi|^2 I
    const double K2[9] = {px * px - th2, px * py, px * pz, px * py, py * py - th2, py * pz, px * pz, py * pz, pz * pz - th2};
    double V[9];
#pragma unroll
    for (int i = 0; i < 9; ++i) {
        const double I = (i % 4 == 0) ? 1.0 : 0.0;
        E.R[i] = I + A * K[i] + B * K2[i];
        V[i] = I + B * K[i] + C * K2[i];
    }
#pragma unroll
    for (int r = 0; r < 3; ++r) E.t[r] = V[3 * r] * d[0] + V[3 * r + 1] * d[1] + V[3 * r + 2] * d[2];
}

// Serial section of one iteration (thread 0 of block 0): assemble H, b from the 29 reduced terms, solve, update
// the pose, decide termination, write the result when done.  Returns the new pose and the done flag.
__device__ __forceinline__ bool solve_and_update(const GicpParams& P, const double* tv, const Pose& T, int it, Pose& Tn) {
    double H[36], b[6];
    {
        int q = 0;
#pragma unroll
        for (int a = 0; a < 6; ++a)
#pragma unroll
            for (int c = a; c < 6; ++c) { H[6 * a + c] = tv[q]; H[6 * c + a] = tv[q]; ++q; }
    }
#pragma unroll
    for (int a = 0; a < 6; ++a) b[a] = tv[21 + a];
    const int n_inl = (int)(tv[28] + 0.5);
    bool done = false;
    int converged = 0, status = FAR_OK;
    Tn = T;
    if (!P.linearize_only) {
        double rhs[6], delta[6];
#pragma unroll
        for (int a = 0; a < 6; ++a) rhs[a] = -b[a];
        if (n_inl < 6 || !chol_solve6(H, rhs, delta)) {
            status = FAR_ERR_DEGENERATE;
            Tn = P.d_init ? *P.d_init : P.init;
            done = true;
        } else {
            Pose E;
            se3_exp(delta, E);
#pragma unroll
            for (int i = 0; i < 3; ++i)
#pragma unroll
                for (int j = 0; j < 3; ++j)
                    Tn.R[3 * i + j] = E.R[3 * i] * T.R[j] + E.R[3 * i + 1] * T.R[3 + j] + E.R[3 * i + 2] * T.R[6 + j];
#pragma unroll
            for (int r = 0; r < 3; ++r)
                Tn.t[r] = (E.R[3 * r] * T.t[0] + E.R[3 * r + 1] * T.t[1] + E.R[3 * r + 2] * T.t[2]) + E.t[r];
            double nrm = 0.0;
#pragma unroll
            for (int a = 0; a < 6; ++a) nrm += delta[a] * delta[a];
            if (nrm <= P.conv_eps * P.conv_eps) { converged = 1; done = true; }   // PAPER.md:100, R13: ||delta||_2 <= eps
        }
    } else {
        done = true;
    }
    if (it + 1 >= P.max_iters) done = true;
    if (done) {
        far_gicp_result_t* out = P.out;
        for (int a = 0; a < 9; ++a) out->pose.R[a] = Tn.R[a];
        for (int a = 0; a < 3; ++a) out->pose.t[a] = Tn.t[a];
        for (int a = 0; a < 36; ++a) out->H[a] = H[a];
        for (int a = 0; a < 6; ++a) out->b[a] = b[a];
        out->chi2 = tv[27];
        out->n_inliers = n_inl;
        out->iters = it + 1;
        out->converged = converged;
        out->status = status;
    }
    return done;
}

// Polls `count` tagged rows starting at `first` (column = lane) and sums them: warp w takes rows w, w + 8, ... in
// increasing order, then the 8 warp sums are added in warp order by warp 0.  Every block must call with all threads.
__device__ __forceinline__ double block_sum_tagged(const uint4* rows, int first, int count, uint32_t tag, int lane, int wib,
                                                   double (*s_red)[TSTRIDE]) {
    double s = 0.0;
    for (int r = wib; r < count; r += GWARPS) s += wait_tagged(rows + (size_t)(first + r) * TSTRIDE + lane, tag);
    s_red[wib][lane] = s;
    __syncthreads();
    double t = 0.0;
    if (wib == 0) {
#pragma unroll
        for (int w8 = 0; w8 < GWARPS; ++w8) t += s_red[w8][lane];
    }
    __syncthreads();
    return t;   // valid in warp 0
}

__global__ void __launch_bounds__(GWARPS * 32, GICP_BLOCKS_PER_SM) gicp_kernel(MapView m, GicpParams P) {
    __shared__ CandList s_list[GWARPS];
    __shared__ double s_terms[GWARPS][TSTRIDE];
    __shared__ double s_red[GWARPS][TSTRIDE];
    __shared__ Corr s_corr[GWARPS];
    __shared__ Src s_src[GWARPS];
    __shared__ Pose s_T;
    __shared__ int s_done;
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const int64_t nwarps = (int64_t)gridDim.x * GWARPS;
    // launch sequence: read by every block at start, advanced by block 0 at the very end (launches on one map are
    // stream-ordered), so every launch has its own tag space without a host-side counter or a kernel argument
    const uint32_t seq = *reinterpret_cast<volatile uint32_t*>(&P.scratch.pub[15].x);
    int64_t n = P.n;
    if (P.d_n) n = min(n, *P.d_n);
    if (threadIdx.x < 12) {
        const Pose& src = P.d_init ? *P.d_init : P.init;
        double vv = threadIdx.x < 9 ? src.R[threadIdx.x] : src.t[threadIdx.x - 9];
        if (threadIdx.x < 9) s_T.R[threadIdx.x] = vv; else s_T.t[threadIdx.x - 9] = vv;
    }
    __syncthreads();
    const int n_groups = (gridDim.x + GROUP - 1) / GROUP;
    const int group = blockIdx.x / GROUP;
    const int group_rows = min(GROUP, (int)gridDim.x - group * GROUP);
    const bool have_scan_cov = P.cov6 != nullptr && P.valid != nullptr && m.cov != nullptr;
    const int rounds = (int)((n + nwarps - 1) / nwarps);      // source points per warp (1 when n <= resident warps)

    // one source point per warp (n <= resident warps, the usual case): the point, its covariance and flag are the same
    // in every iteration, so they are fetched once and stay in registers -- one memory level less per iteration.
    // Lane l < 8 of warp 0 holds the point of warp l (phase A0), lanes 8..14 of every warp its own covariance and flag.
    const bool resident = rounds == 1;
    float sx0 = 0.f, sy0 = 0.f, sz0 = 0.f, cin0 = 0.f;
    if (resident) {
        if (wib == 0 && lane < GWARPS) {
            const int64_t i = (int64_t)blockIdx.x * GWARPS + lane;
            sx0 = sy0 = sz0 = __int_as_float(0x7FC00000);     // NaN: no point
            if (i < n) {
                const float* sp = P.scan + i * P.stride;
                sx0 = __ldg(sp); sy0 = __ldg(sp + 1); sz0 = __ldg(sp + 2);
            }
        }
        const int64_t i = (int64_t)blockIdx.x * GWARPS + wib;
        if (i < n && have_scan_cov) {
            if (lane >= 8 && lane < 14) cin0 = __ldg(P.cov6 + 6 * i + (lane - 8));
            if (lane == 14) cin0 = (float)__ldg(P.valid + i);
        }
    }

    for (int it = 0; it < P.max_iters; ++it) {
        const uint32_t tag = (seq << 10) | (uint32_t)(it + 1);
        double acc = 0.0;                                     // warp 0, lane t < 29: term t of this block
        for (int rd = 0; rd < rounds; ++rd) {
            // ---- phase A0 (Eq. 2, A1): 8 lanes of warp 0 transform the block's 8 source points with the accumulated pose
            // (R11) and take their voxel indices: one instruction stream for 8 points instead of 8 redundant warps ------
            if (wib == 0 && lane < GWARPS) {
                float sx = sx0, sy = sy0, sz = sz0;
                if (!resident) {
                    const int64_t i = (int64_t)rd * nwarps + (int64_t)blockIdx.x * GWARPS + lane;
                    sx = sy = sz = __int_as_float(0x7FC00000);
                    if (i < n) {
                        const float* sp = P.scan + i * P.stride;
                        sx = __ldg(sp); sy = __ldg(sp + 1); sz = __ldg(sp + 2);
                    }
                }
                Src o;
                o.ok = 0;
                o.p[0] = o.p[1] = o.p[2] = 0.f;
                o.k[0] = o.k[1] = o.k[2] = 0;
                if (isfinite(sx) && isfinite(sy) && isfinite(sz)) {
                    transform_point(s_T, sx, sy, sz, o.p);
                    o.ok = voxel_index(o.p[0], o.p[1], o.p[2], m.voxel, o.k) ? 1 : 0;
                }
                s_src[lane] = o;
            }
            __syncthreads();
            // ---- phase A (A8): one warp per source point -> correspondence record ---------------------------------
            const int64_t i = (int64_t)rd * nwarps + (int64_t)blockIdx.x * GWARPS + wib;
            int flags = 0;
            if (i < n) {
                float cin = cin0;
                if (!resident && have_scan_cov) {
                    // the source covariance does not depend on the search: lanes 8..13 fetch it now, lane 14 its flag
                    if (lane >= 8 && lane < 14) cin = __ldg(P.cov6 + 6 * i + (lane - 8));
                    if (lane == 14) cin = (float)__ldg(P.valid + i);
                }
                const Src src = s_src[wib];
                const float pf[3] = {src.p[0], src.p[1], src.p[2]};
                const int k[3] = {src.k[0], src.k[1], src.k[2]};
                {
                    if (src.ok) {
                        // kNN-search, k = 1
                        float rx, ry, rz;
                        const Best best = warp_nearest(m, pf[0], pf[1], pf[2], k, lane, s_list[wib], rx, ry, rz);
                        if (best.id != NO_ID && !(best.d2 > P.tau2)) {    // adaptive-threshold gate
                            // lanes 0..5 fetch Sigma_r, lane 6 its flag: one memory level
                            if (have_scan_cov) {
                                if (lane < 6) cin = __ldg(m.cov + (size_t)best.ref * 6 + lane);
                                if (lane == 6) cin = (float)__ldg(m.cov_ok + best.ref);
                            }
                            const bool full = have_scan_cov && __shfl_sync(FULL, cin, 6) != 0.f && __shfl_sync(FULL, cin, 14) != 0.f;
                            Corr& c = s_corr[wib];
                            if (lane < 6) c.cr[lane] = cin;
                            if (lane >= 8 && lane < 14) c.cs[lane - 8] = cin;
                            if (lane == 16) { c.p[0] = pf[0]; c.p[1] = pf[1]; c.p[2] = pf[2]; c.r[0] = rx; c.r[1] = ry; c.r[2] = rz; }
                            flags = full ? 3 : 1;
                        }
                    }
                }
            }
            if (lane == 0) s_corr[wib].flags = flags;
            __syncthreads();
            // ---- phase B (A9): 8 lanes of warp 0 linearise the block's 8 correspondences together --------------------
            if (wib == 0) {
                if (lane < GWARPS) {
                    const Corr c = s_corr[lane];
                    double* terms = s_terms[lane];
                    if (c.flags & 1) {
                        const double p[3] = {(double)c.p[0], (double)c.p[1], (double)c.p[2]};
                        const double r[3] = {(double)c.r[0], (double)c.r[1], (double)c.r[2]};
                        correspondence_terms(s_T, p, r, (c.flags & 2) != 0, c.cs, c.cr, P.kernel, P.kappa, terms);
                    } else {
#pragma unroll
                        for (int t = 0; t < NTERMS; ++t) terms[t] = 0.0;
                    }
                }
                __syncwarp();
                if (lane < NTERMS) {
#pragma unroll
                    for (int w8 = 0; w8 < GWARPS; ++w8) acc += s_terms[w8][lane];
                }
            }
            if (rd + 1 < rounds) __syncthreads();             // the records are rewritten by the next round
        }
        // ---- A10: block row -> group of 32 blocks -> grid, tagged words, every level summed in a fixed order --------
        if (wib == 0) put_tagged(P.scratch.rows + (size_t)blockIdx.x * TSTRIDE + lane, lane < NTERMS ? acc : 0.0, tag);
        if (blockIdx.x % GROUP == 0) {   // group leader: fold the group's rows into one
            const double t = block_sum_tagged(P.scratch.rows, group * GROUP, group_rows, tag, lane, wib, s_red);
            if (wib == 0) put_tagged(P.scratch.grows + (size_t)group * TSTRIDE + lane, t, tag);
            if (blockIdx.x == 0) {       // block 0: final sum, solve, publish
                const double t2 = block_sum_tagged(P.scratch.grows, 0, n_groups, tag, lane, wib, s_red);
                if (wib == 0) s_terms[0][lane] = t2;
                __syncthreads();
                if (threadIdx.x == 0) {
                    Pose Tn;
                    const bool done = solve_and_update(P, s_terms[0], s_T, it, Tn);
#pragma unroll
                    for (int a = 0; a < 9; ++a) put_tagged(P.scratch.pub + a, Tn.R[a], tag);
#pragma unroll
                    for (int a = 0; a < 3; ++a) put_tagged(P.scratch.pub + 9 + a, Tn.t[a], tag);
                    put_tagged(P.scratch.pub + 12, done ? 1.0 : 0.0, tag);
                }
            }
        }
        // ---- grid-wide wait for the new pose: all blocks are co-resident (cooperative launch) -----------------------
        __syncthreads();                                      // phase B / the sums have finished reading s_T, s_terms
        if (wib == 0) {
            // ONE lane per block polls the `done` word (written last); only when it carries this iteration's tag do the
            // other twelve lanes fetch their words (each still self-validating).  740 pollers on one line instead of
            // 9,620 on two: the solver's stores no longer queue behind the poll traffic in that L2 slice (on some B200s
            // of the pool the publish hop cost 3.5 us instead of 1.1 us with every lane polling).
            double vv = 0.0;
            if (lane == NPUB - 1) {
                uint4 w = load_tagged(P.scratch.pub + lane);
                while (w.y != tag || w.w != tag) {
                    __nanosleep(200);       // back off: the waiters must not crowd out the few blocks still working
                    w = load_tagged(P.scratch.pub + lane);
                }
                vv = __longlong_as_double((long long)(((unsigned long long)w.z << 32) | w.x));
            }
            __syncwarp();
            if (lane < NPUB - 1) vv = wait_tagged(P.scratch.pub + lane, tag);
            if (lane < 9) s_T.R[lane] = vv;
            else if (lane < 12) s_T.t[lane - 9] = vv;
            else if (lane == 12) s_done = vv != 0.0 ? 1 : 0;
        }
        __syncthreads();
        if (s_done) break;
    }
    // every block has read `seq` before it could pass the first grid-wide wait, which block 0 is now behind
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        uint32_t next = (seq + 1u) & 0x3FFFFFu;
        if (next == 0u) {
            // wrap-around of the 22-bit sequence (once per 4 M launches): wipe the block and group rows so that no word
            // written 4 M launches ago can be mistaken for a current one (every row this launch needed has been read: the
            // solve came after them; the published words are rewritten by every launch and stay).  Tag 0 is never used
            const size_t words = (size_t)(P.scratch.pub - P.scratch.rows);
            for (size_t w = 0; w < words; ++w) P.scratch.rows[w] = make_uint4(0u, 0u, 0u, 0u);
            next = 1u;
        }
        __threadfence();
        *reinterpret_cast<volatile uint32_t*>(&P.scratch.pub[15].x) = next;
    }
}

}  // namespace far

extern "C" {

void far_gicp_default_options(far_gicp_options_t* o) {
    if (!o) return;
    o->kernel = FAR_KERNEL_CAUCHY;
    o->conv_eps = 5e-3;
    o->tau_mult = 3.0;
    o->kappa_div = 3.0;
}

static int gicp_launch(const far_map_t* map, const float* d_scan, const float* d_cov6, const uint8_t* d_valid, int64_t n,
                       const int64_t* d_n, int stride, const far_pose_t* hpose, const far_pose_t* d_pose, double sigma,
                       int max_iters, int linearize_only, const far_gicp_options_t* opts, far_gicp_result_t* d_out,
                       void* stream) {
    if (!map || !d_out || n < 0 || (n > 0 && !d_scan) || (stride != 3 && stride != 4) || max_iters < 1 || max_iters > MAX_ITERS_LIMIT || (!hpose && !d_pose))
        return FAR_ERR_ARG;
    far_gicp_options_t o;
    if (opts) o = *opts; else far_gicp_default_options(&o);
    if (o.kernel < 0 || o.kernel > 2 || !(sigma > 0.0)) return FAR_ERR_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    GicpParams P;
    memset(&P, 0, sizeof(P));
    P.scan = d_scan; P.cov6 = d_cov6; P.valid = d_valid; P.n = n; P.d_n = d_n; P.stride = stride;
    if (hpose) memcpy(&P.init, hpose, sizeof(Pose));
    P.d_init = (const Pose*)d_pose;
    const double tau = o.tau_mult * sigma;
    P.tau2 = tau * tau;
    P.kappa = sigma / o.kappa_div;
    P.conv_eps = o.conv_eps;
    P.kernel = o.kernel; P.max_iters = max_iters; P.linearize_only = linearize_only;
    P.scratch.rows = reinterpret_cast<uint4*>(map->d_gicp_partials);
    P.scratch.grows = P.scratch.rows + (size_t)map->gicp_max_grid * TSTRIDE;
    P.scratch.pub = P.scratch.grows + (size_t)MAX_GROUPS * TSTRIDE;
    P.out = d_out;
    int64_t grid = map->gicp_max_grid;
    const int64_t need = (n + GWARPS - 1) / GWARPS;
    if (need < grid) grid = need;
    if (grid < 1) grid = 1;
    MapView view = map->view;
    void* args[] = {(void*)&view, (void*)&P};
    {
        far::LaunchScope ls_("gicp_kernel", st);
        FAR_CUDA(cudaLaunchCooperativeKernel((const void*)gicp_kernel, dim3((unsigned)grid), dim3(GWARPS * 32), args, 0, st));
    }
    return FAR_OK;
}

int far_gicp_linearize(const far_map_t* map, const float* d_scan, const float* d_cov6, const uint8_t* d_valid, int64_t n,
                       int stride, const far_pose_t* pose, double sigma, const far_gicp_options_t* opts,
                       far_gicp_result_t* d_out, void* stream) {
    return gicp_launch(map, d_scan, d_cov6, d_valid, n, nullptr, stride, pose, nullptr, sigma, 1, 1, opts, d_out, stream);
}

int far_gicp_register(const far_map_t* map, const float* d_scan, const float* d_cov6, const uint8_t* d_valid, int64_t n,
                      int stride, const far_pose_t* init_pose, double sigma, int max_iters, const far_gicp_options_t* opts,
                      far_gicp_result_t* d_out, void* stream) {
    return gicp_launch(map, d_scan, d_cov6, d_valid, n, nullptr, stride, init_pose, nullptr, sigma, max_iters, 0, opts, d_out,
                       stream);
}

int far_gicp_register_dev(const far_map_t* map, const float* d_scan, const float* d_cov6, const uint8_t* d_valid,
                          const int64_t* d_n, int64_t n_max, int stride, const far_pose_t* d_init_pose, double sigma,
                          int max_iters, const far_gicp_options_t* opts, far_gicp_result_t* d_out, void* stream) {
    if (!d_n || !d_init_pose) return FAR_ERR_ARG;
    return gicp_launch(map, d_scan, d_cov6, d_valid, n_max, d_n, stride, nullptr, d_init_pose, sigma, max_iters, 0, opts, d_out,
                       stream);
}

// n from the device, initial pose from the host as a kernel argument (saves far_frontend_process a pageable
// 96-byte upload per frame)
int far_gicp_register_dn(const far_map_t* map, const float* d_scan, const float* d_cov6, const uint8_t* d_valid,
                         const int64_t* d_n, int64_t n_max, int stride, const far_pose_t* init_pose, double sigma, int max_iters,
                         const far_gicp_options_t* opts, far_gicp_result_t* d_out, void* stream) {
    if (!d_n || !init_pose) return FAR_ERR_ARG;
    return gicp_launch(map, d_scan, d_cov6, d_valid, n_max, d_n, stride, init_pose, nullptr, sigma, max_iters, 0, opts, d_out, stream);
}


}  // extern "C"

namespace far {
static size_t gicp_scratch_bytes(int max_grid) { return ((size_t)(max_grid + MAX_GROUPS) * TSTRIDE + 16) * sizeof(uint4); }

// called once from far_map_create: sizes the cooperative grid and allocates the reduction scratch
int gicp_setup(far_map* map) {
    int per_sm = 0;
    FAR_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, gicp_kernel, GWARPS * 32, 0));
    if (per_sm < 1) per_sm = 1;
    map->gicp_max_grid = map->sm_count * per_sm;
    if (map->gicp_max_grid > GROUP * MAX_GROUPS) map->gicp_max_grid = GROUP * MAX_GROUPS;
    const size_t bytes = gicp_scratch_bytes(map->gicp_max_grid);
    FAR_CUDA(cudaMalloc((void**)&map->d_gicp_partials, bytes));
    FAR_CUDA(cudaMemset(map->d_gicp_partials, 0, bytes));     // tag 0 is never used by a launch
    const uint32_t one = 1u;                                   // launch sequence starts at 1 (pub[15].x)
    FAR_CUDA(cudaMemcpy(reinterpret_cast<uint4*>(map->d_gicp_partials) + (size_t)(map->gicp_max_grid + MAX_GROUPS) * TSTRIDE + 15,
                        &one, sizeof(one), cudaMemcpyHostToDevice));
    return FAR_OK;
}
}  // namespace far
