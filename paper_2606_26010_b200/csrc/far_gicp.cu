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
//   phase A  one warp per source point, no block barrier before it: the warp transforms its point itself (FP64), and
//            what the previous iteration learnt stays in registers -- the source point and its covariance, the 27 table
//            lookups (valid as long as the transformed point stays in its voxel: the map does not change during a
//            registration) and the previous nearest neighbour, whose distance to the new position bounds the search: a
//            neighbour voxel is read only if its distance lower bound does not exceed it (exact, ties included).  From
//            the second iteration on a search is usually one sweep over the point's own voxel, served by L1;
//   phase B  the block's 8 correspondences are linearised by 8 lanes of warp 0 at once (one FP64 instruction stream for
//            8 points: the FP64 pipe, not the issue slots, is what a per-warp linearisation would exhaust), column by
//            column so that the live set fits the 48 registers five co-resident blocks per SM leave;
//   reduce   the 29 unique terms of (H, b, chi2, n) go block -> group of 32 blocks -> grid as TAGGED rows: every
//            value travels as two 8-byte words {value half, tag} (tag = launch sequence and iteration), so a consumer
//            just polls the rows it needs -- no fence, no ticket atomics -- and sums them in a fixed order
//            (deterministic, no floating-point atomics);
//   solve    warp 0 of block 0: 6x6 Cholesky with one row per lane (shuffles, no local memory), SE(3) exponential by
//            series, pose update and stop test in FP64; thirteen lanes publish one tagged word each; one lane per block
//            polls the `done` word with a short back-off, then twelve lanes fetch the pose.
// The host is not involved until it reads the result.
//
// Tagged words and the PTX memory model: a word is written with st.relaxed.gpu.v2.u64 and read with ld.relaxed.gpu.v2.u64.
// PTX treats a vector access as one scalar access per element, and an aligned 64-bit scalar access is single-copy atomic,
// so each element {32 value bits, 32 tag bits} is observed whole or not at all; a reader accepts a value only when BOTH
// elements carry the tag it waits for.  No ordering between different words is assumed anywhere.
#include <cstring>

#include "far_internal.h"

using namespace far;

namespace far {

constexpr int GWARPS = 8;        // warps per block = correspondences linearised together in phase B
constexpr int NTERMS = 29;       // 21 (H upper triangle) + 6 (b) + chi2 + inlier count
constexpr int TSTRIDE = 32;      // row length of the tagged rows in global memory
constexpr int SSTRIDE = 33;      // row length of the per-correspondence term rows in shared memory (no bank conflicts)

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
    const double* d_sigma;      // nullable: tau2 = (tau_mult sigma)^2 and kappa = sigma / kappa_div from the DEVICE value
    double tau_mult, kappa_div;
    int kernel, max_iters, linearize_only;
    GicpScratch scratch;
    far_gicp_result_t* out;
};

__device__ __forceinline__ void put_tagged(uint4* dst, double v, uint32_t tag) {
    const unsigned long long b = (unsigned long long)__double_as_longlong(v), t = (unsigned long long)tag << 32;
    asm volatile("st.relaxed.gpu.global.v2.u64 [%0], {%1, %2};" ::"l"(dst), "l"(t | (b & 0xFFFFFFFFull)), "l"(t | (b >> 32)) : "memory");
}

// one attempt: true (and the value) iff both elements carry `tag`
__device__ __forceinline__ bool load_tagged(const uint4* src, uint32_t tag, double& v) {
    unsigned long long a, b;
    asm volatile("ld.relaxed.gpu.global.v2.u64 {%0, %1}, [%2];" : "=l"(a), "=l"(b) : "l"(src) : "memory");
    v = __longlong_as_double((long long)((b << 32) | (a & 0xFFFFFFFFull)));
    return (uint32_t)(a >> 32) == tag && (uint32_t)(b >> 32) == tag;
}

// spins until both halves carry `tag` (volatile asm: the compiler must neither hoist the load nor assume the loop ends)
__device__ __forceinline__ double wait_tagged(const uint4* src, uint32_t tag) {
    double v;
    while (!load_tagged(src, tag, v)) {}
    return v;
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

// A9 for one correspondence: the 29 terms, written straight into the correspondence's row of shared memory.  Ordered so
// that few values are live at a time: S row by row -> M -> (M, Md, w) -> one column of X = M [p]x and of Y = [p]x^T X at
// a time.  H = w J^T M J with J = [-I | A], A = [p]x:  [[M, -X], [-X^T, Y]];  b = w J^T M d = w [-Md ; A^T Md].
__device__ __forceinline__ void correspondence_terms(const Pose& T, const Corr& c, int kernel, double kappa, double* terms) {
    const double px = (double)c.p[0], py = (double)c.p[1], pz = (double)c.p[2];
    const double d0 = (double)c.r[0] - px, d1 = (double)c.r[1] - py, d2 = (double)c.r[2] - pz;   // Eq. 3
    double M[6] = {1.0, 0.0, 0.0, 1.0, 0.0, 1.0};                        // SA fallback: Sigma_r = I, Sigma_s = 0
    if (c.flags & 2) {
        // S = Sigma_r + R Sigma_s R^T   (Eq. 4): row i of R Sigma_s, then its products with rows j >= i of R
        const double s0 = c.cs[0], s1 = c.cs[1], s2 = c.cs[2], s3 = c.cs[3], s4 = c.cs[4], s5 = c.cs[5];
        double S[6];
        {
            const double a = T.R[0], b = T.R[1], e = T.R[2];
            const double u0 = a * s0 + b * s1 + e * s2, u1 = a * s1 + b * s3 + e * s4, u2 = a * s2 + b * s4 + e * s5;
            S[0] = (double)c.cr[0] + (u0 * T.R[0] + u1 * T.R[1] + u2 * T.R[2]);
            S[1] = (double)c.cr[1] + (u0 * T.R[3] + u1 * T.R[4] + u2 * T.R[5]);
            S[2] = (double)c.cr[2] + (u0 * T.R[6] + u1 * T.R[7] + u2 * T.R[8]);
        }
        {
            const double a = T.R[3], b = T.R[4], e = T.R[5];
            const double u0 = a * s0 + b * s1 + e * s2, u1 = a * s1 + b * s3 + e * s4, u2 = a * s2 + b * s4 + e * s5;
            S[3] = (double)c.cr[3] + (u0 * T.R[3] + u1 * T.R[4] + u2 * T.R[5]);
            S[4] = (double)c.cr[4] + (u0 * T.R[6] + u1 * T.R[7] + u2 * T.R[8]);
        }
        {
            const double a = T.R[6], b = T.R[7], e = T.R[8];
            const double u0 = a * s0 + b * s1 + e * s2, u1 = a * s1 + b * s3 + e * s4, u2 = a * s2 + b * s4 + e * s5;
            S[5] = (double)c.cr[5] + (u0 * T.R[6] + u1 * T.R[7] + u2 * T.R[8]);
        }
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
    terms[0] = w * M[0];  terms[1] = w * M[1];  terms[2] = w * M[2];
    terms[6] = w * M[3];  terms[7] = w * M[4];  terms[11] = w * M[5];
    terms[21] = -w * Md0; terms[22] = -w * Md1; terms[23] = -w * Md2;
    terms[24] = w * (pz * Md1 - py * Md2);
    terms[25] = w * (px * Md2 - pz * Md0);
    terms[26] = w * (py * Md0 - px * Md1);
    terms[27] = w * e2;
    terms[28] = 1.0;
    // column 0 of X = M A:  X[r][0] = M[r][1] pz - M[r][2] py;   Y[i][0] = (A^T X)[i][0]
    {
        const double x0 = M[1] * pz - M[2] * py, x1 = M[3] * pz - M[4] * py, x2 = M[4] * pz - M[5] * py;
        terms[3] = -w * x0; terms[8] = -w * x1; terms[12] = -w * x2;
        terms[15] = w * (pz * x1 - py * x2);                               // Y00
    }
    // column 1:  X[r][1] = M[r][2] px - M[r][0] pz
    {
        const double x0 = M[2] * px - M[0] * pz, x1 = M[4] * px - M[1] * pz, x2 = M[5] * px - M[2] * pz;
        terms[4] = -w * x0; terms[9] = -w * x1; terms[13] = -w * x2;
        terms[16] = w * (pz * x1 - py * x2);                               // Y01
        terms[18] = w * (px * x2 - pz * x0);                               // Y11
    }
    // column 2:  X[r][2] = M[r][0] py - M[r][1] px
    {
        const double x0 = M[0] * py - M[1] * px, x1 = M[1] * py - M[3] * px, x2 = M[2] * py - M[4] * px;
        terms[5] = -w * x0; terms[10] = -w * x1; terms[14] = -w * x2;
        terms[17] = w * (pz * x1 - py * x2);                               // Y02
        terms[19] = w * (px * x2 - pz * x0);                               // Y12
        terms[20] = w * (py * x0 - px * x1);                               // Y22
    }
}

// A6 with what earlier iterations learnt: `cnt` / `bucket` are the warp's 27 lookups for voxel k (lane l < 27), `bound0`
// an upper bound of the answer's d2 (+inf if none): the distance to a stored point that lies in the 27 voxels.  A voxel is
// read only if its distance lower bound does not exceed the bound; without a bound the point's own voxel is swept first
// to get one.  Exactly the (d2, id) minimum of R6: a skipped voxel holds only points strictly farther than the bound.
__device__ __forceinline__ Best nearest_bounded(const MapView& m, float qx, float qy, float qz, const int k[3], int lane,
                                                uint32_t cnt, uint32_t bucket, double bound0, CandList& L, float& rx, float& ry, float& rz) {
    const double INF = __longlong_as_double(0x7FF0000000000000ll);
    Best best;
    best.d2 = INF; best.id = NO_ID; best.ref = 0;
    float bx = 0.f, by = 0.f, bz = 0.f;
    double bound = bound0;
    const bool have_bound = bound0 < INF;
    if (!have_bound) {
        const uint32_t c_cnt = __shfl_sync(FULL, cnt, 13), c_bucket = __shfl_sync(FULL, bucket, 13);
        for (uint32_t j = lane; j < c_cnt; j += 32) {
            const uint32_t ref = c_bucket * (uint32_t)m.cap + j;
            const float4 p = __ldg(m.points + ref);
            const double d2 = dist2(qx, qy, qz, p.x, p.y, p.z);
            const uint32_t id = __float_as_uint(p.w);
            if (better(d2, id, best)) { best.d2 = d2; best.id = id; best.ref = ref; bx = p.x; by = p.y; bz = p.z; }
        }
        bound = warp_min_nonneg(best.d2);
    }
    uint32_t c2 = 0;
    if (lane < 27 && cnt > 0 && (have_bound || lane != 13)) {
        const double lb = (lane == 13) ? 0.0 : voxel_lower_bound(qx, qy, qz, k, m.voxel, lane / 9 - 1, (lane / 3) % 3 - 1, lane % 3 - 1);
        if (lb <= bound) c2 = cnt;
    }
    const unsigned surv = __ballot_sync(FULL, c2 > 0);
    if ((surv & ~(1u << 13)) == 0) {
        // the usual case from the second iteration on: no neighbour voxel can hold a nearer point.  With a bound the own
        // voxel is still to be swept (one step: cap <= 64 points, two lanes' worth at most); without, it was swept above
        if (surv) {
            const uint32_t c_cnt = __shfl_sync(FULL, c2, 13), c_bucket = __shfl_sync(FULL, bucket, 13);
            for (uint32_t j = lane; j < c_cnt; j += 32) {
                const uint32_t ref = c_bucket * (uint32_t)m.cap + j;
                const float4 p = __ldg(m.points + ref);
                const double d2 = dist2(qx, qy, qz, p.x, p.y, p.z);
                const uint32_t id = __float_as_uint(p.w);
                if (better(d2, id, best)) { best.d2 = d2; best.id = id; best.ref = ref; bx = p.x; by = p.y; bz = p.z; }
            }
        }
        const int w = warp_argmin(best.d2, best.id);
        best.d2 = __shfl_sync(FULL, best.d2, w);
        best.id = __shfl_sync(FULL, best.id, w);
        best.ref = __shfl_sync(FULL, best.ref, w);
        rx = __shfl_sync(FULL, bx, w); ry = __shfl_sync(FULL, by, w); rz = __shfl_sync(FULL, bz, w);
        return best;
    }
    const int total = cand_build(L, c2, bucket, lane);
    CandIter ci;
    ci.before = 0;
    for (int j = lane, step = 0; j < total; j += 32, ++step) {
        const uint32_t ref = cand_next(L, ci, step, j, lane, m.cap);
        const float4 p = __ldg(m.points + ref);
        const double d2 = dist2(qx, qy, qz, p.x, p.y, p.z);
        const uint32_t id = __float_as_uint(p.w);
        if (better(d2, id, best)) { best.d2 = d2; best.id = id; best.ref = ref; bx = p.x; by = p.y; bz = p.z; }
    }
    __syncwarp();
    const int w = warp_argmin(best.d2, best.id);
    best.d2 = __shfl_sync(FULL, best.d2, w);
    best.id = __shfl_sync(FULL, best.id, w);
    best.ref = __shfl_sync(FULL, best.ref, w);
    rx = __shfl_sync(FULL, bx, w); ry = __shfl_sync(FULL, by, w); rz = __shfl_sync(FULL, bz, w);
    return best;
}

// 6x6 Cholesky solve H x = rhs by one warp: lane i < 6 owns row i (H is read from the packed upper triangle `tv` in
// shared memory as it is needed) and rhs_i; every lane returns all of x.  The factor's row i lives in lane i's registers
// with the RECIPROCAL pivot in place of L_ii (the pivot itself is never needed again); rows talk through shuffles, so
// nothing spills and the six pivots are the only serial chain.  One rsqrt per pivot.  false if H is not positive
// definite.  All 32 lanes must call (lanes >= 6 compute on row 5's data and are ignored).
__device__ __forceinline__ bool warp_chol_solve6(const double* tv, double rhs, int lane, double x[6]) {
    const int i = min(lane, 5);
    double l[6];
    bool ok = true;
#pragma unroll
    for (int j = 0; j < 6; ++j) {
        const int a = min(i, j), c = max(i, j);
        double acc = tv[a * 6 - a * (a - 1) / 2 + (c - a)];                        // H_ij
#pragma unroll
        for (int k = 0; k < j; ++k) acc -= l[k] * __shfl_sync(FULL, l[k], j);     // H_ij - sum_k L_ik L_jk
        const double piv = __shfl_sync(FULL, acc, j);
        ok = ok && piv > 0.0 && isfinite(piv);
        const double inv = rsqrt(piv);
        l[j] = (lane == j) ? inv : acc * inv;                                      // lanes i < j hold garbage: never read
    }
    // forward: y_k = (rhs_k - sum_{j<k} L_kj y_j) / L_kk, finished on lane k and broadcast
    double y = rhs, z = 0.0;
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        const double yk = __shfl_sync(FULL, y * l[k], k);
        if (lane == k) z = yk;
        y -= l[k] * yk;                                                             // lanes i > k; others unused
    }
    // backward: x_k = (y_k - sum_{i>k} L_ik x_i) / L_kk; L_ik sits in lane i, which sends its product to lane k
#pragma unroll
    for (int k = 5; k >= 0; --k) {
        const double xk = __shfl_sync(FULL, z * l[k], k);
        x[k] = xk;
#pragma unroll
        for (int q = 0; q < k; ++q) {
            const double c = __shfl_sync(FULL, l[q] * xk, k);                      // lane k's L_kq x_k, for lane q
            if (lane == q) z -= c;
        }
    }
    return ok;
}

// coefficients of the SE(3) exponential: A = sin t / t, B = (1 - cos t) / t^2, C = (t - sin t) / t^3.  Series in t^2 up
// to t^10 below 0.1 rad (remainder < 1e-21 relative: a Gauss-Newton increment is always that small unless the initial
// guess is far off), the closed forms above.
__device__ __forceinline__ void exp_coefficients(double th2, double& A, double& B, double& C) {
    if (th2 < 0.01) {
        A = 1.0 + th2 * (-1.0 / 6.0 + th2 * (1.0 / 120.0 + th2 * (-1.0 / 5040.0 + th2 * (1.0 / 362880.0 + th2 * (-1.0 / 39916800.0)))));
        B = 0.5 + th2 * (-1.0 / 24.0 + th2 * (1.0 / 720.0 + th2 * (-1.0 / 40320.0 + th2 * (1.0 / 3628800.0 + th2 * (-1.0 / 479001600.0)))));
        C = 1.0 / 6.0 + th2 * (-1.0 / 120.0 + th2 * (1.0 / 5040.0 + th2 * (-1.0 / 362880.0 + th2 * (1.0 / 39916800.0 + th2 * (-1.0 / 6227020800.0)))));
    } else {
        const double th = sqrt(th2);
        double sn, cs;
        sincos(th, &sn, &cs);
        const double ith2 = 1.0 / th2;
        A = sn / th; B = (1.0 - cs) * ith2; C = (th - sn) * ith2 / th;
    }
}

// Serial section of one iteration, run by warp 0 of block 0 (all 32 lanes call): H, b from the 29 reduced terms `tv`
// (shared memory), solve, SE(3) exponential, pose update, stop test; lanes 0..12 publish one tagged word each, the result
// struct is written lane-parallel when the registration ends.
__device__ __forceinline__ void solve_and_publish(const GicpParams& P, const double* tv, const Pose& T, int it, int lane, uint32_t tag) {
    // index of H[a][c] (a <= c) in the packed upper triangle
    auto tri = [](int a, int c) { return a * 6 - a * (a - 1) / 2 + (c - a); };
    const double rhs = -tv[21 + min(lane, 5)];
    const int n_inl = (int)(tv[28] + 0.5);
    double delta[6];
    const bool solved = warp_chol_solve6(tv, rhs, lane, delta);
    bool done = false;
    int converged = 0, status = FAR_OK;
    // the element of the new pose this lane owns: lanes 0..8 R (row-major), 9..11 t
    double mine = 0.0;
    const int r = lane < 9 ? lane / 3 : lane - 9, cidx = lane % 3;
    if (P.linearize_only) {
        done = true;
        if (lane < 9) mine = T.R[lane]; else if (lane < 12) mine = T.t[lane - 9];
    } else if (n_inl < 6 || !solved) {
        status = FAR_ERR_DEGENERATE;
        done = true;
        const Pose& I0 = P.d_init ? *P.d_init : P.init;
        if (lane < 9) mine = I0.R[lane]; else if (lane < 12) mine = I0.t[lane - 9];
    } else {
        const double px = delta[3], py = delta[4], pz = delta[5];
        const double th2 = px * px + py * py + pz * pz;
        double A, B, C;
        exp_coefficients(th2, A, B, C);
        // row r of E.R = I + A K + B K^2 and of V = I + B K + C K^2, K = [phi]x, K^2 = phi phi^T - |phi|^2 I
        const double ph[3] = {px, py, pz};
        const double pr = r == 0 ? px : (r == 1 ? py : pz);
        double er[3], vr[3];
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            const double k2 = pr * ph[j] - (j == r ? th2 : 0.0);
            // K[r][j]: (0,1) -pz (0,2) py (1,0) pz (1,2) -px (2,0) -py (2,1) px
            double kk = 0.0;
            if (r == 0) kk = j == 1 ? -pz : (j == 2 ? py : 0.0);
            else if (r == 1) kk = j == 0 ? pz : (j == 2 ? -px : 0.0);
            else kk = j == 0 ? -py : (j == 1 ? px : 0.0);
            const double id = j == r ? 1.0 : 0.0;
            er[j] = id + A * kk + B * k2;
            vr[j] = id + B * kk + C * k2;
        }
        if (lane < 9) mine = er[0] * T.R[cidx] + er[1] * T.R[3 + cidx] + er[2] * T.R[6 + cidx];
        else if (lane < 12) mine = (er[0] * T.t[0] + er[1] * T.t[1] + er[2] * T.t[2]) + (vr[0] * delta[0] + vr[1] * delta[1] + vr[2] * delta[2]);
        double nrm = 0.0;
#pragma unroll
        for (int a = 0; a < 6; ++a) nrm += delta[a] * delta[a];
        if (nrm <= P.conv_eps * P.conv_eps) { converged = 1; done = true; }   // PAPER.md:100, R13: ||delta||_2 <= eps
    }
    if (it + 1 >= P.max_iters) done = true;
    if (lane < 12) put_tagged(P.scratch.pub + lane, mine, tag);
    if (done) {
        far_gicp_result_t* out = P.out;
        if (lane < 9) out->pose.R[lane] = mine; else if (lane < 12) out->pose.t[lane - 9] = mine;
        for (int a = lane; a < 36; a += 32) { const int i = a / 6, j = a % 6; out->H[a] = tv[i <= j ? tri(i, j) : tri(j, i)]; }
        if (lane < 6) out->b[lane] = tv[21 + lane];
        if (lane == 6) out->chi2 = tv[27];
        if (lane == 7) { out->n_inliers = n_inl; out->iters = it + 1; out->converged = converged; out->status = status; }
    }
    if (lane == 12) put_tagged(P.scratch.pub + 12, done ? 1.0 : 0.0, tag);
}

// Polls `count` tagged rows starting at `first` (column = lane) and sums them: warp w takes rows w, w + 8, ... in
// increasing order, then the 8 warp sums are added in warp order by warp 0.  Every block must call with all threads.
__device__ __forceinline__ double block_sum_tagged(const uint4* rows, int first, int count, uint32_t tag, int lane, int wib,
                                                   double (*s_red)[TSTRIDE]) {
    // a warp's rows are requested together before the first is examined: they arrive within a microsecond of each other,
    // and one L2 round trip per row would be most of the reduction
    constexpr int POLL = 4;
    double s = 0.0;
    for (int r0 = wib; r0 < count; r0 += GWARPS * POLL) {
        double v[POLL];
        unsigned pending = 0;
#pragma unroll
        for (int u = 0; u < POLL; ++u) {
            const int r = r0 + u * GWARPS;
            v[u] = 0.0;
            if (r < count && !load_tagged(rows + (size_t)(first + r) * TSTRIDE + lane, tag, v[u])) pending |= 1u << u;
        }
#pragma unroll
        for (int u = 0; u < POLL; ++u) {
            if (pending & (1u << u)) v[u] = wait_tagged(rows + (size_t)(first + r0 + u * GWARPS) * TSTRIDE + lane, tag);
            s += v[u];                                       // fixed order: rows ascending
        }
    }
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

// what a warp keeps about its source point from one iteration to the next (shared memory: 30-cycle reads instead of
// registers the FP64 linearisation needs)
struct WarpState {
    float s[3];       // the source point (sensor frame)
    float pr[3];      // previous nearest neighbour
    int kr[3];        // its voxel
    int kp[3];        // voxel of the transformed point at the last table walk
    uint32_t pref;    // reference of the previous nearest neighbour
};

__global__ void __launch_bounds__(GWARPS * 32, GICP_BLOCKS_PER_SM) gicp_kernel(const __grid_constant__ MapView m, const __grid_constant__ GicpParams P) {
    __shared__ CandList s_list[GWARPS];
    __shared__ double s_terms[GWARPS][SSTRIDE];
    __shared__ double s_red[GWARPS][TSTRIDE];
    __shared__ Corr s_corr[GWARPS];
    __shared__ WarpState s_state[GWARPS];
    __shared__ Pose s_T;
    __shared__ int s_done;
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const int nwarps = (int)gridDim.x * GWARPS;
    // launch sequence: read by every block at start, advanced by block 0 at the very end (launches on one map are
    // stream-ordered), so every launch has its own tag space without a host-side counter or a kernel argument
    const uint32_t seq = *reinterpret_cast<volatile uint32_t*>(&P.scratch.pub[15].x);
    int n = (int)P.n;
    if (P.d_n) n = (int)min((int64_t)n, *P.d_n);
    if (threadIdx.x < 12) {
        const Pose& src = P.d_init ? *P.d_init : P.init;
        double vv = threadIdx.x < 9 ? src.R[threadIdx.x] : src.t[threadIdx.x - 9];
        if (threadIdx.x < 9) s_T.R[threadIdx.x] = vv; else s_T.t[threadIdx.x - 9] = vv;
    }
    const bool have_scan_cov = P.cov6 != nullptr && P.valid != nullptr && m.cov != nullptr;
    double tau2 = P.tau2, kappa = P.kappa;
    if (P.d_sigma) {                                          // frame graph: sigma is part of the device-side frame parameters
        const double sg = *P.d_sigma;
        tau2 = (P.tau_mult * sg) * (P.tau_mult * sg);
        kappa = sg / P.kappa_div;
    }
    const int rounds = (n + nwarps - 1) / nwarps;             // source points per warp (1 when n <= resident warps)
    const double INF = __longlong_as_double(0x7FF0000000000000ll);

    // one source point per warp (n <= resident warps, the usual case): everything that does not depend on the pose is
    // fetched once and kept across iterations -- the point in shared memory, its covariance in lanes 8..13 and its flag
    // in lane 14.  What an iteration learns is kept too: the voxel the transformed point fell into with its 27 lookups
    // (lane l < 27: count, bucket), the nearest neighbour (reference, coordinates) and, in lanes 0..6, that
    // neighbour's covariance and flag.
    const bool resident = rounds == 1;
    WarpState& ws = s_state[wib];
    float cin0 = 0.f;
    if (resident) {
        const int i = (int)blockIdx.x * GWARPS + wib;
        if (i < n) {
            if (lane < 3) ws.s[lane] = __ldg(P.scan + (int64_t)i * P.stride + lane);
            if (have_scan_cov) {
                if (lane >= 8 && lane < 14) cin0 = __ldg(P.cov6 + 6 * (int64_t)i + (lane - 8));
                if (lane == 14) cin0 = (float)__ldg(P.valid + i);
            }
        }
    }
    __syncthreads();
    uint32_t have = 0;                    // bit 0: the 27 lookups are those of voxel ws.kp; bit 1: ws.pr / ws.pref are set
    uint32_t pcnt = 0, pbucket = NO_BUCKET;
    float cinr = 0.f;

    for (int it = 0; it < P.max_iters; ++it) {
        const uint32_t tag = (seq << 10) | (uint32_t)(it + 1);
        double acc = 0.0;                                     // warp 0, lane t < 29: term t of this block
        for (int rd = 0; rd < rounds; ++rd) {
            // ---- phase A (Eq. 2, A1, A6, A8): one warp per source point -> correspondence record ---------------------
            const int i = rd * nwarps + (int)blockIdx.x * GWARPS + wib;
            int flags = 0;
            if (i < n) {
                float sx, sy, sz, cin = cin0;
                if (resident) {
                    sx = ws.s[0]; sy = ws.s[1]; sz = ws.s[2];
                } else {
                    const float* sp = P.scan + (int64_t)i * P.stride;
                    sx = __ldg(sp); sy = __ldg(sp + 1); sz = __ldg(sp + 2);
                    if (have_scan_cov) {
                        if (lane >= 8 && lane < 14) cin = __ldg(P.cov6 + 6 * (int64_t)i + (lane - 8));
                        if (lane == 14) cin = (float)__ldg(P.valid + i);
                    }
                    have = 0;
                }
                float pf[3];
                int k[3];
                bool ok = false;
                if (isfinite(sx) && isfinite(sy) && isfinite(sz)) {
                    transform_point(s_T, sx, sy, sz, pf);                       // accumulated pose on the ORIGINAL point (R11)
                    ok = voxel_index(pf[0], pf[1], pf[2], m.voxel, k);
                }
                if (ok) {
                    // the 27 lookups: reused while the point stays in its voxel
                    if (!((have & 1u) && k[0] == ws.kp[0] && k[1] == ws.kp[1] && k[2] == ws.kp[2])) {
                        probe27_regs(m, k, lane, pcnt, pbucket);
                        __syncwarp();
                        if (lane < 3) ws.kp[lane] = k[lane];
                        have |= 1u;
                    }
                    // the previous nearest neighbour bounds the search if it is one of this search's candidates
                    double bound = INF;
                    uint32_t pref = 0xFFFFFFFFu;
                    if (have & 2u) {
                        pref = ws.pref;
                        if (abs(ws.kr[0] - k[0]) <= 1 && abs(ws.kr[1] - k[1]) <= 1 && abs(ws.kr[2] - k[2]) <= 1)
                            bound = dist2(pf[0], pf[1], pf[2], ws.pr[0], ws.pr[1], ws.pr[2]);
                    }
                    // kNN-search, k = 1
                    float rx, ry, rz;
                    const Best best = nearest_bounded(m, pf[0], pf[1], pf[2], k, lane, pcnt, pbucket, bound, s_list[wib], rx, ry, rz);
                    if (best.id != NO_ID) {
                        // Sigma_r (lanes 0..5) and its flag (lane 6): one memory level, skipped if the neighbour is the old one
                        if (have_scan_cov && best.ref != pref) {
                            if (lane < 6) cinr = __ldg(m.cov + (size_t)best.ref * 6 + lane);
                            if (lane == 6) cinr = (float)__ldg(m.cov_ok + best.ref);
                        }
                        __syncwarp();
                        if (best.ref != pref && lane == 0) {
                            ws.pr[0] = rx; ws.pr[1] = ry; ws.pr[2] = rz; ws.pref = best.ref;
                            int kr[3];
                            voxel_index(rx, ry, rz, m.voxel, kr);                 // a stored point: always valid
                            ws.kr[0] = kr[0]; ws.kr[1] = kr[1]; ws.kr[2] = kr[2];
                        }
                        have |= 2u;
                        if (!(best.d2 > tau2)) {                                 // adaptive-threshold gate
                            const bool full = have_scan_cov && __shfl_sync(FULL, cinr, 6) != 0.f && __shfl_sync(FULL, cin, 14) != 0.f;
                            Corr& c = s_corr[wib];
                            if (lane < 6) c.cr[lane] = cinr;
                            if (lane >= 8 && lane < 14) c.cs[lane - 8] = cin;
                            if (lane == 16) { c.p[0] = pf[0]; c.p[1] = pf[1]; c.p[2] = pf[2]; c.r[0] = rx; c.r[1] = ry; c.r[2] = rz; }
                            flags = full ? 3 : 1;
                        }
                    } else {
                        have &= ~2u;
                    }
                    __syncwarp();
                }
            }
            if (lane == 0) s_corr[wib].flags = flags;
            __syncthreads();
            // ---- phase B (A9): 8 lanes of warp 0 linearise the block's 8 correspondences together --------------------
            if (wib == 0) {
                if (lane < GWARPS) {
                    double* terms = s_terms[lane];
                    if (s_corr[lane].flags & 1) {
                        correspondence_terms(s_T, s_corr[lane], P.kernel, kappa, terms);
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
            const int group = blockIdx.x / GROUP, n_groups = (gridDim.x + GROUP - 1) / GROUP;
            const int group_rows = min(GROUP, (int)gridDim.x - group * GROUP);
            const double t = block_sum_tagged(P.scratch.rows, group * GROUP, group_rows, tag, lane, wib, s_red);
            if (wib == 0) put_tagged(P.scratch.grows + (size_t)group * TSTRIDE + lane, t, tag);
            if (blockIdx.x == 0) {       // block 0: final sum, solve, publish
                const double t2 = block_sum_tagged(P.scratch.grows, 0, n_groups, tag, lane, wib, s_red);
                if (wib == 0) {
                    s_red[0][lane] = t2;
                    __syncwarp();
                    solve_and_publish(P, s_red[0], s_T, it, lane, tag);
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
                while (!load_tagged(P.scratch.pub + lane, tag, vv)) __nanosleep(40);    // back off: do not crowd out the blocks still working
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

}  // extern "C"

int far::gicp_launch(const far_map_t* map, const float* d_scan, const float* d_cov6, const uint8_t* d_valid, int64_t n,
                     const int64_t* d_n, int stride, const far_pose_t* hpose, const far_pose_t* d_pose, double sigma,
                     const double* d_sigma, int max_iters, int linearize_only, const far_gicp_options_t* opts, far_gicp_result_t* d_out,
                     void* stream) {
    if (!map || !d_out || n < 0 || n > 0x7FFFFFFFll / 8 || (n > 0 && !d_scan) || (stride != 3 && stride != 4) || max_iters < 1 || max_iters > MAX_ITERS_LIMIT || (!hpose && !d_pose))
        return FAR_ERR_ARG;
    far_gicp_options_t o;
    if (opts) o = *opts; else far_gicp_default_options(&o);
    if (o.kernel < 0 || o.kernel > 2 || (!d_sigma && !(sigma > 0.0))) return FAR_ERR_ARG;
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
    P.d_sigma = d_sigma; P.tau_mult = o.tau_mult; P.kappa_div = o.kappa_div;
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

extern "C" {

int far_gicp_linearize(const far_map_t* map, const float* d_scan, const float* d_cov6, const uint8_t* d_valid, int64_t n,
                       int stride, const far_pose_t* pose, double sigma, const far_gicp_options_t* opts,
                       far_gicp_result_t* d_out, void* stream) {
    return far::gicp_launch(map, d_scan, d_cov6, d_valid, n, nullptr, stride, pose, nullptr, sigma, nullptr, 1, 1, opts, d_out, stream);
}

int far_gicp_register(const far_map_t* map, const float* d_scan, const float* d_cov6, const uint8_t* d_valid, int64_t n,
                      int stride, const far_pose_t* init_pose, double sigma, int max_iters, const far_gicp_options_t* opts,
                      far_gicp_result_t* d_out, void* stream) {
    return far::gicp_launch(map, d_scan, d_cov6, d_valid, n, nullptr, stride, init_pose, nullptr, sigma, nullptr, max_iters, 0, opts,
                            d_out, stream);
}

int far_gicp_register_dev(const far_map_t* map, const float* d_scan, const float* d_cov6, const uint8_t* d_valid,
                          const int64_t* d_n, int64_t n_max, int stride, const far_pose_t* d_init_pose, double sigma,
                          int max_iters, const far_gicp_options_t* opts, far_gicp_result_t* d_out, void* stream) {
    if (!d_n || !d_init_pose) return FAR_ERR_ARG;
    return far::gicp_launch(map, d_scan, d_cov6, d_valid, n_max, d_n, stride, nullptr, d_init_pose, sigma, nullptr, max_iters, 0, opts,
                            d_out, stream);
}

// n from the device, initial pose from the host as a kernel argument (saves far_frontend_process a pageable
// 96-byte upload per frame)
int far_gicp_register_dn(const far_map_t* map, const float* d_scan, const float* d_cov6, const uint8_t* d_valid,
                         const int64_t* d_n, int64_t n_max, int stride, const far_pose_t* init_pose, double sigma, int max_iters,
                         const far_gicp_options_t* opts, far_gicp_result_t* d_out, void* stream) {
    if (!d_n || !init_pose) return FAR_ERR_ARG;
    return far::gicp_launch(map, d_scan, d_cov6, d_valid, n_max, d_n, stride, init_pose, nullptr, sigma, nullptr, max_iters, 0, opts, d_out, stream);
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
