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
// B200 design: a registration is a few thousand source points, i.e. latency- and issue-bound, never bandwidth-bound, so
// the whole Gauss-Newton loop is ONE persistent cooperative kernel and an iteration is organised to keep both the
// instruction count per scheduler and the serial chain short (round 2 profile: with a warp per point, 10 warps per
// scheduler each issued ~950 instructions per iteration -- 5-7 us -- and seven warps of a block waited at a barrier
// while 8 lanes of the eighth linearised):
//   groups   GLANES = 16 lanes per source point, two points per warp; points are dealt round-robin over the blocks of the
//            grid (ONE block of GWARPS = 20 warps = 640 threads per SM, 40 points per block and round), so a 5,000-point
//            scan is served in one round by 148 blocks and the per-point scalar work (transform, voxel index, bounds)
//            is issued once per 2 points;
//   search   what the previous iteration learnt stays with the group: the 27 table lookups (lane g keeps neighbours g and
//            g + 16; valid while the transformed point stays in its voxel: the map does not change during a
//            registration) and the previous nearest neighbour, whose distance to the new position bounds the search: a
//            neighbour voxel is read only if its distance lower bound does not exceed it (exact, ties included).  From the
//            second iteration on a search is usually one sweep over the point's own voxel, served by L1;
//   A9       every group linearises its own correspondence at once -- no block barrier, no serial section: the six
//            entries of Sigma_r + R Sigma_s R^T one per lane, M = S^-1, M d and the weight in every lane, and the 29
//            terms of (H, b, chi2, n) as ONE uniform expression  coef (u[a] u[b] - u[c] u[d])  over a small vector u
//            = (M, M d, p, 0, 1, e2, X) in shared memory with a constant index table (TERM_SLOTS = 3 term columns per
//            lane: entries g, g + 16 < 24, then 24 + g), so the lanes do not diverge;
//   reduce   lane-wise across the 2 groups of a warp (shuffles), across the warps of the block (shared memory), then
//            block -> group of 16 blocks -> grid as TAGGED rows: every value travels as two 8-byte words {value half,
//            tag} (tag = launch sequence and iteration), so a consumer just polls the rows it needs -- no fence, no
//            ticket atomics -- and sums them in a fixed order (deterministic, no floating-point atomics);
//   solve    warp 0 of block 0: 6x6 Gauss-Jordan on [H | -b] with one row per lane (pivots = those of Cholesky, so
//            "not positive definite" is detected identically; six reciprocals are the serial chain, no square roots, no
//            substitution passes), SE(3) exponential by series, pose update and stop test in FP64; thirteen lanes publish
//            one tagged word each; one lane per block polls the `done` word with a short back-off, then twelve lanes
//            fetch the pose.
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

constexpr int GLANES = 16;                // lanes per source point (8 or 16)
constexpr int GWARPS = 20;                // warps per block
constexpr int GTHREADS = GWARPS * 32;
constexpr int GPTS = GTHREADS / GLANES;   // source points per block and round
constexpr int NBR_PER_LANE = (27 + GLANES - 1) / GLANES;   // neighbour voxels a lane looks after: l = g + GLANES j
constexpr int SWEEP_U = 32 / GLANES;                      // candidate loads in flight per lane: 32 per group and round trip
constexpr int TERM_SLOTS = (24 + GLANES - 1) / GLANES + 1;               // term columns per lane: entries g, g + GLANES, .. < 24, then 24 + g
constexpr int GICP_BLOCKS_PER_SM = 1;
// (a row of the reduction carries 29 terms: 21 of H's upper triangle, 6 of b, chi2, inlier count; 3 columns idle)
constexpr int TSTRIDE = 32;               // row length of the tagged rows in global memory
constexpr int GROUP = 16;                 // blocks per first-level reduction group (one hop over all 148 rows measured 2 % slower)
constexpr int MAX_GROUPS = 64;
constexpr int NPUB = 13;                  // published words: R[9], t[3], done
constexpr int MAX_ITERS_LIMIT = 1000;     // the iteration index shares the 32-bit tag with the launch sequence

// device scratch of one map: [max_grid] block rows, [MAX_GROUPS] group rows, the published pose
struct GicpScratch {
    uint4* rows;      // [max_grid][TSTRIDE]
    uint4* grows;     // [MAX_GROUPS][TSTRIDE]
    uint4* pub;       // [16]: 13 published words; pub[15].x = launch sequence of this map (device-resident)
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
    int sm_count;
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
    if (kernel == FAR_KERNEL_CAUCHY) { const double k2 = kappa * kappa; return k2 / (k2 + e2); }   // Eq. 5 as IRLS weight (R9): 1 / (1 + e2 / kappa^2), one division
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

// ---- A9 as one uniform expression ---------------------------------------------------------------------------------------
// H = w J^T M J with J = [-I | A], A = [p]x:  [[M, -X], [-X^T, Y]], X = M A, Y = A^T X;  b = w J^T M d = w [-Md ; A^T Md].
// Every one of the 29 terms is coef * (u[a] u[b] - u[c] u[d]) over the group's vector
//   u = (M0..M5 | Md0..Md2 | px py pz | 0 | 1 | e2 | X00 X01 X02 X10 .. X22)          (24 doubles in shared memory)
// with coef in {+w, -w, 1}.  Lane g of a group evaluates entries g, 8 + g, 16 + g of the first round (the nine X, which it
// also stores into u, the six M, -Md, A^T Md, chi2, n) and entry g of the second (the six Y, which need X).  An entry packs
// a | b << 5 | c << 10 | d << 15 | coef << 20 | (1 + X index) << 22; c_term_store maps the entry to its column in the
// 29-term row (H upper triangle row-wise, b, chi2, n).
constexpr int U_MD = 6, U_P = 9, U_ZERO = 12, U_ONE = 13, U_E2 = 14, U_X = 15, U_LEN = 24;
constexpr uint32_t term_enc(int a, int b, int c, int d, int coef, int xs) {
    return (uint32_t)a | ((uint32_t)b << 5) | ((uint32_t)c << 10) | ((uint32_t)d << 15) | ((uint32_t)coef << 20) | ((uint32_t)xs << 22);
}
constexpr int sym3(int r, int c) { return r == c ? (r == 0 ? 0 : (r == 1 ? 3 : 5)) : (r + c == 1 ? 1 : (r + c == 2 ? 2 : 4)); }
constexpr int COEF_W = 0, COEF_MW = 1, COEF_ONE = 2;
// X[r][0] = M[r][1] pz - M[r][2] py;  X[r][1] = M[r][2] px - M[r][0] pz;  X[r][2] = M[r][0] py - M[r][1] px
constexpr uint32_t x_enc(int r, int c) {
    return c == 0 ? term_enc(sym3(r, 1), U_P + 2, sym3(r, 2), U_P + 1, COEF_MW, 1 + 3 * r + c)
         : c == 1 ? term_enc(sym3(r, 2), U_P + 0, sym3(r, 0), U_P + 2, COEF_MW, 1 + 3 * r + c)
                  : term_enc(sym3(r, 0), U_P + 1, sym3(r, 1), U_P + 0, COEF_MW, 1 + 3 * r + c);
}
constexpr uint32_t plain_enc(int a, int coef) { return term_enc(a, U_ONE, U_ZERO, U_ZERO, coef, 0); }
constexpr int XI(int r, int c) { return U_X + 3 * r + c; }
__constant__ uint32_t c_term_enc[32] = {
    // round 1, slot 0
    x_enc(0, 0), x_enc(0, 1), x_enc(0, 2), x_enc(1, 0), x_enc(1, 1), x_enc(1, 2), x_enc(2, 0), x_enc(2, 1),
    // slot 1
    x_enc(2, 2), plain_enc(0, COEF_W), plain_enc(1, COEF_W), plain_enc(2, COEF_W), plain_enc(3, COEF_W), plain_enc(4, COEF_W),
    plain_enc(5, COEF_W), plain_enc(U_MD + 0, COEF_MW),
    // slot 2:  b_phi = w A^T Md = w (pz Md1 - py Md2, px Md2 - pz Md0, py Md0 - px Md1)
    plain_enc(U_MD + 1, COEF_MW), plain_enc(U_MD + 2, COEF_MW),
    term_enc(U_P + 2, U_MD + 1, U_P + 1, U_MD + 2, COEF_W, 0), term_enc(U_P + 0, U_MD + 2, U_P + 2, U_MD + 0, COEF_W, 0),
    term_enc(U_P + 1, U_MD + 0, U_P + 0, U_MD + 1, COEF_W, 0), plain_enc(U_E2, COEF_W), plain_enc(U_ONE, COEF_ONE),
    term_enc(U_ZERO, U_ZERO, U_ZERO, U_ZERO, COEF_ONE, 0),
    // round 2 (slot 3):  Y[0][j] = pz X[1][j] - py X[2][j];  Y[1][j] = px X[2][j] - pz X[0][j];  Y[2][j] = py X[0][j] - px X[1][j]
    term_enc(U_P + 2, XI(1, 0), U_P + 1, XI(2, 0), COEF_W, 0), term_enc(U_P + 2, XI(1, 1), U_P + 1, XI(2, 1), COEF_W, 0),
    term_enc(U_P + 2, XI(1, 2), U_P + 1, XI(2, 2), COEF_W, 0), term_enc(U_P + 0, XI(2, 1), U_P + 2, XI(0, 1), COEF_W, 0),
    term_enc(U_P + 0, XI(2, 2), U_P + 2, XI(0, 2), COEF_W, 0), term_enc(U_P + 1, XI(0, 2), U_P + 0, XI(1, 2), COEF_W, 0),
    term_enc(U_ZERO, U_ZERO, U_ZERO, U_ZERO, COEF_ONE, 0), term_enc(U_ZERO, U_ZERO, U_ZERO, U_ZERO, COEF_ONE, 0)};
__constant__ uint8_t c_term_store[32] = {
    3, 4, 5, 8, 9, 10, 12, 13,
    14, 0, 1, 2, 6, 7, 11, 21,
    22, 23, 24, 25, 26, 27, 28, 29,
    15, 16, 17, 18, 19, 20, 30, 31};

// group-wide arg-min over (d2, id) (lanes of `gmask`): returns the warp lane holding the winner
__device__ __forceinline__ int group_argmin(unsigned gmask, double d2, uint32_t id) {
    const unsigned long long bits = (unsigned long long)__double_as_longlong(d2);
    const uint32_t hi = (uint32_t)(bits >> 32), lo = (uint32_t)bits;
    const uint32_t mhi = __reduce_min_sync(gmask, hi);
    bool c = hi == mhi;
    const uint32_t mlo = __reduce_min_sync(gmask, c ? lo : 0xFFFFFFFFu);
    c = c && lo == mlo;
    unsigned b = __ballot_sync(gmask, c);
    if (b & (b - 1)) {      // more than one lane holds the minimal d2: lowest id wins (R6)
        const uint32_t mid = __reduce_min_sync(gmask, c ? id : 0xFFFFFFFFu);
        c = c && id == mid;
        b = __ballot_sync(gmask, c);
    }
    return __ffs(b) - 1;
}

__device__ __forceinline__ double group_min_nonneg(unsigned gmask, double d2) {
    const unsigned long long bits = (unsigned long long)__double_as_longlong(d2);
    const uint32_t hi = (uint32_t)(bits >> 32), lo = (uint32_t)bits;
    const uint32_t mhi = __reduce_min_sync(gmask, hi);
    const uint32_t mlo = __reduce_min_sync(gmask, hi == mhi ? lo : 0xFFFFFFFFu);
    return __longlong_as_double((long long)(((unsigned long long)mhi << 32) | mlo));
}

__device__ __forceinline__ double shfl_d(unsigned mask, double v, int src) { return __shfl_sync(mask, v, src); }

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

// 6x6 solve H x = rhs by one warp, Gauss-Jordan on the augmented rows: lane i < 6 owns row i of [H | rhs] (H from the
// packed upper triangle `tv`); step k broadcasts row k, every other row eliminates column k, row k is normalised.  H is
// symmetric positive definite in every non-degenerate registration, so no row exchange is needed and pivot k is exactly
// the k-th pivot of the Cholesky factorisation squared: "some pivot <= 0" is the same verdict.  Serial chain: six
// reciprocals.  Every lane returns all of x; false if H is not positive definite.  All 32 lanes must call.
__device__ __forceinline__ bool warp_solve6(const double* tv, double rhs, int lane, double x[6]) {
    const int i = min(lane, 5);
    double a[7];
#pragma unroll
    for (int j = 0; j < 6; ++j) {
        const int lo = min(i, j), hi = max(i, j);
        a[j] = tv[lo * 6 - lo * (lo - 1) / 2 + (hi - lo)];
    }
    a[6] = rhs;
    bool ok = true;
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        double pk[7];
#pragma unroll
        for (int j = k; j < 7; ++j) pk[j] = __shfl_sync(FULL, a[j], k);
        const double piv = pk[k];
        ok = ok && piv > 0.0 && isfinite(piv);
        const double r = 1.0 / piv;
        const double f = a[k] * r;
#pragma unroll
        for (int j = k; j < 7; ++j) a[j] = (lane == k) ? pk[j] * r : a[j] - f * pk[j];
    }
#pragma unroll
    for (int j = 0; j < 6; ++j) x[j] = __shfl_sync(FULL, a[6], j);
    return ok;
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
    const bool solved = warp_solve6(tv, rhs, lane, delta);
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

// Polls `count` tagged rows starting at `first` (column = lane) and sums them: warp w takes rows w, w + GWARPS, ... in
// increasing order, then the warp sums are added in warp order by warp 0.  Every thread of the block must call.
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

// what a group keeps in shared memory about its source point (read once per iteration; the registers go to the FP64 work)
struct PointState {
    float s[3];       // the source point (sensor frame)
    float pr[3];      // previous nearest neighbour
    int kr[3];        // its voxel
};

__global__ void __launch_bounds__(GTHREADS, GICP_BLOCKS_PER_SM) gicp_kernel(const __grid_constant__ MapView m, const __grid_constant__ GicpParams P) {
    __shared__ double s_u[GPTS][U_LEN];
    __shared__ double s_part[GWARPS][32];
    __shared__ double s_red[GWARPS][TSTRIDE];
    __shared__ float s_cs[GPTS][6];
    __shared__ uint32_t s_lb[GPTS][28], s_lo[GPTS][28];       // a group's surviving voxels: bucket, first candidate index
    __shared__ PointState s_state[GPTS];
    __shared__ Pose s_T;
    __shared__ int s_done;
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const int gl = lane & (GLANES - 1), base = lane & ~(GLANES - 1);
    const unsigned gmask = (GLANES == 32 ? 0xFFFFFFFFu : ((1u << GLANES) - 1u)) << base;
    const int slot = threadIdx.x / GLANES;                    // the group's index in the block
    // launch sequence: read by every block at start, advanced by block 0 at the very end (launches on one map are
    // stream-ordered), so every launch has its own tag space without a host-side counter or a kernel argument
    const uint32_t seq = *reinterpret_cast<volatile uint32_t*>(&P.scratch.pub[15].x);
    int n = (int)P.n;
    if (P.d_n) n = (int)min((int64_t)n, *P.d_n);
    // blocks in use: one per SM while that holds the scan (fewer rows to reduce), never fewer than a warp's worth of
    // points per block; the others leave at once (nothing below synchronises through the grid's size)
    int G = (int)gridDim.x;
    {
        const int per_sm = (n + P.sm_count * GPTS - 1) / (P.sm_count * GPTS);
        G = min(G, max(1, P.sm_count * max(per_sm, 1)));
        G = min(G, max(1, (n + 3) / 4));
    }
    if ((int)blockIdx.x >= G) return;
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
    // points are dealt round-robin over the blocks: point i of round rd sits in block i mod grid, so a scan smaller than
    // the grid's capacity (the usual case) spreads evenly over all SMs instead of filling the first blocks
    const int per_round = G * GPTS;
    const int rounds = (n + per_round - 1) / per_round;
    const bool resident = rounds <= 1;                        // every group keeps ONE point for the whole registration
    const double INF = __longlong_as_double(0x7FF0000000000000ll);
    const double dv = (double)m.voxel;
    PointState& ps = s_state[slot];
    double* u = s_u[slot];

    // what does not depend on the pose is fetched once: the point and its covariance (shared memory), its flag (lane 6)
    float cin = 0.f;                                          // lane 6: Sigma_s valid
    auto load_point = [&](int i) {
        if (gl < 3) ps.s[gl] = __ldg(P.scan + (int64_t)i * P.stride + gl);
        cin = 0.f;
        if (have_scan_cov) {
            if (gl < 6) s_cs[slot][gl] = __ldg(P.cov6 + 6 * (int64_t)i + gl);
            if (gl == 6) cin = (float)__ldg(P.valid + i);
        }
        __syncwarp(gmask);
    };
    {
        const int i = slot * G + (int)blockIdx.x;
        if (resident && i < n) load_point(i);
    }
    __syncthreads();
    // what an iteration learns: the voxel the transformed point fell into with its 27 lookups (lane g: neighbours g + 8 j;
    // counts packed one byte each), the nearest neighbour (reference; coordinates and voxel in shared memory) and, in lanes
    // 0..6, that neighbour's covariance and flag
    // this lane's entries of the term table, fetched once (a lane-dependent index into constant memory is replayed per
    // distinct address: 16 replays per access inside the loop)
    uint32_t enc[TERM_SLOTS];
#pragma unroll
    for (int q = 0; q < TERM_SLOTS; ++q) enc[q] = c_term_enc[(q < TERM_SLOTS - 1 ? q * GLANES + gl : 24 + (gl & 7)) & 31];
    uint32_t have = 0;                    // bit 0: the lookups are those of voxel kp; bit 1: the previous neighbour is set
    int kp0 = 0, kp1 = 0, kp2 = 0;
    uint32_t pcnt[NBR_PER_LANE], pbk[NBR_PER_LANE], pref = 0xFFFFFFFFu;
#pragma unroll
    for (int j = 0; j < NBR_PER_LANE; ++j) { pcnt[j] = 0; pbk[j] = NO_BUCKET; }
    float cinr = 0.f;

    for (int it = 0; it < P.max_iters; ++it) {
        const uint32_t tag = (seq << 10) | (uint32_t)(it + 1);
        double acc[TERM_SLOTS];                                     // this lane's term columns, summed over its points
#pragma unroll
        for (int q = 0; q < TERM_SLOTS; ++q) acc[q] = 0.0;
        for (int rd = 0; rd < rounds; ++rd) {
            const int i = (rd * GPTS + slot) * G + (int)blockIdx.x;
            if (i >= n) continue;                                   // group-uniform: everything below uses gmask
            if (!resident) { load_point(i); have = 0; }
            // ---- Eq. 2: the accumulated pose on the ORIGINAL point (R11); lane g computes coordinate g mod 3 ---------
            const float sx = ps.s[0], sy = ps.s[1], sz = ps.s[2];
            const int r3 = gl % 3;
            float pmine;
            {
                double a = __dadd_rn(__dmul_rn(s_T.R[3 * r3 + 0], (double)sx), __dmul_rn(s_T.R[3 * r3 + 1], (double)sy));
                a = __dadd_rn(a, __dmul_rn(s_T.R[3 * r3 + 2], (double)sz));
                a = __dadd_rn(a, s_T.t[r3]);
                pmine = __double2float_rn(a);
            }
            // A1 of my coordinate
            const float fq = floorf(__fdiv_rn(pmine, m.voxel));
            const bool inr = fq >= -1048576.0f && fq < 1048576.0f;
            const int kmine = inr ? (int)fq : 0;
            const float pfx = __shfl_sync(gmask, pmine, base), pfy = __shfl_sync(gmask, pmine, base + 1), pfz = __shfl_sync(gmask, pmine, base + 2);
            const int k0 = __shfl_sync(gmask, kmine, base), k1 = __shfl_sync(gmask, kmine, base + 1), k2 = __shfl_sync(gmask, kmine, base + 2);
            const bool ok = isfinite(sx) && isfinite(sy) && isfinite(sz) && ((__ballot_sync(gmask, inr) >> base) & 7u) == 7u;
            if (!ok) continue;
            // ---- the 27 lookups: reused while the point stays in its voxel ---------------------------------------------
            if (!((have & 1u) && k0 == kp0 && k1 == kp1 && k2 == kp2)) {
                // home entries of this lane's neighbours first, all in flight together (a walk beyond the home slot is rare)
                unsigned long long key[NBR_PER_LANE];
                Entry he[NBR_PER_LANE];
                uint32_t hs[NBR_PER_LANE];
#pragma unroll
                for (int j = 0; j < NBR_PER_LANE; ++j) {
                    const int l = gl + GLANES * j;
                    const int nx = k0 + l / 9 - 1, ny = k1 + (l / 3) % 3 - 1, nz = k2 + l % 3 - 1;
                    const bool in = l < 27 && index_in_range(nx) && index_in_range(ny) && index_in_range(nz);
                    key[j] = in ? pack_key(nx, ny, nz) : KEY_EMPTY;
                    hs[j] = hash_key(key[j]) & m.mask;
                    he[j].key = KEY_EMPTY; he[j].bucket = NO_BUCKET; he[j].cr = 0;
                    if (in) he[j] = load_entry(m.table, hs[j]);
                }
#pragma unroll
                for (int j = 0; j < NBR_PER_LANE; ++j) {
                    pcnt[j] = 0; pbk[j] = NO_BUCKET;
                    if (key[j] != KEY_EMPTY && he[j].key != KEY_EMPTY) {
                        Entry e = he[j];
                        const uint32_t reach = entry_reach(e.cr);
                        for (uint32_t d = 0;; ++d) {                           // find_voxel from the loaded home entry on
                            if (e.key == key[j]) {
                                const uint32_t c = entry_count(e.cr);
                                if (c && e.bucket < BUCKET_PENDING) { pcnt[j] = c; pbk[j] = e.bucket; }
                                break;
                            }
                            if (d >= reach) break;
                            e = load_entry(m.table, (hs[j] + d + 1) & m.mask);
                            if (e.key == KEY_EMPTY) break;
                        }
                    }
                }
                kp0 = k0; kp1 = k1; kp2 = k2;
                have |= 1u;
            }
            // ---- A6: bounded search (k = 1) ----------------------------------------------------------------
            Best best;
            best.d2 = INF; best.id = NO_ID; best.ref = 0;
            float bx = 0.f, by = 0.f, bz = 0.f;
            auto consider = [&](const float4& p, uint32_t ref) {
                const double d2 = dist2(pfx, pfy, pfz, p.x, p.y, p.z);
                const uint32_t id = __float_as_uint(p.w);
                if (better(d2, id, best)) { best.d2 = d2; best.id = id; best.ref = ref; bx = p.x; by = p.y; bz = p.z; }
            };
            // the previous nearest neighbour bounds the search if it is one of this search's candidates
            double bound = INF;
            uint32_t pref_seen = 0xFFFFFFFFu;
            if (have & 2u) {
                pref_seen = pref;
                if (abs(ps.kr[0] - k0) <= 1 && abs(ps.kr[1] - k1) <= 1 && abs(ps.kr[2] - k2) <= 1)
                    bound = dist2(pfx, pfy, pfz, ps.pr[0], ps.pr[1], ps.pr[2]);
            }
            // without one, the point's own voxel (neighbour 13) is swept first to get a bound
            bool own_swept = false;
            if (!(bound < INF)) {
                const uint32_t c = __shfl_sync(gmask, pcnt[13 / GLANES], base + 13 % GLANES), b = __shfl_sync(gmask, pbk[13 / GLANES], base + 13 % GLANES);
                for (uint32_t j0 = 0; j0 < c; j0 += SWEEP_U * GLANES) {
                    float4 p[SWEEP_U];
#pragma unroll
                    for (int t = 0; t < SWEEP_U; ++t) if (j0 + t * GLANES + gl < c) p[t] = __ldg(m.points + b * (uint32_t)m.cap + j0 + t * GLANES + gl);
#pragma unroll
                    for (int t = 0; t < SWEEP_U; ++t) if (j0 + t * GLANES + gl < c) consider(p[t], b * (uint32_t)m.cap + j0 + t * GLANES + gl);
                }
                bound = group_min_nonneg(gmask, best.d2);
                own_swept = true;
            }
            {
                // squared face gaps of the point inside its voxel, pulled in by the fp32 key-rounding margin (far_common.cuh)
                double lo2[3], hi2[3];
                const double q[3] = {(double)pfx, (double)pfy, (double)pfz};
                const int kk[3] = {k0, k1, k2};
#pragma unroll
                for (int a = 0; a < 3; ++a) {
                    const double margin = (double)(abs(kk[a]) + 2) * dv * 9.5367431640625e-07;   // 2^-20
                    const double lo = fmax(q[a] - (double)kk[a] * dv - margin, 0.0);
                    const double hi = fmax((double)(kk[a] + 1) * dv - q[a] - margin, 0.0);
                    lo2[a] = lo * lo; hi2[a] = hi * hi;
                }
                // a voxel is read only if its distance lower bound does not exceed the bound (a skipped voxel holds only
                // strictly farther points).  The survivors' points are swept as ONE flattened list per group -- compact
                // (bucket, first candidate) pairs in shared memory, built with one packed scan over the 8 lanes -- so that
                // candidate q goes to lane q mod GLANES and 32 loads per group are in flight whatever the voxels' sizes
                uint32_t sc[NBR_PER_LANE];
                uint32_t nsurv = 0, tsum = 0;
#pragma unroll
                for (int j = 0; j < NBR_PER_LANE; ++j) {
                    const int l = gl + GLANES * j;
                    const uint32_t c = pcnt[j];
                    sc[j] = 0;
                    if (l < 27 && c > 0 && !(l == 13 && own_swept)) {
                        const int ox = l / 9 - 1, oy = (l / 3) % 3 - 1, oz = l % 3 - 1;
                        double lb = 0.0;
                        lb += ox < 0 ? lo2[0] : (ox > 0 ? hi2[0] : 0.0);
                        lb += oy < 0 ? lo2[1] : (oy > 0 ? hi2[1] : 0.0);
                        lb += oz < 0 ? lo2[2] : (oz > 0 ? hi2[2] : 0.0);
                        if (lb <= bound) { sc[j] = c; ++nsurv; tsum += c; }
                    }
                }
                const uint32_t packed = (nsurv << 16) | tsum;
                uint32_t incl = packed;
#pragma unroll
                for (int d = 1; d < GLANES; d <<= 1) {
                    const uint32_t o = __shfl_up_sync(gmask, incl, d, GLANES);
                    if (gl >= d) incl += o;
                }
                const uint32_t total = __shfl_sync(gmask, incl, base + GLANES - 1) & 0xFFFFu;
                uint32_t pos = (incl - packed) >> 16, off = (incl - packed) & 0xFFFFu;
                uint32_t* lb_ = s_lb[slot];
                uint32_t* lo_ = s_lo[slot];
#pragma unroll
                for (int j = 0; j < NBR_PER_LANE; ++j) {
                    if (sc[j]) {
                        lb_[pos] = pbk[j];
                        lo_[pos] = off;
                        off += sc[j]; ++pos;
                    }
                }
                if (gl == GLANES - 1) lo_[pos] = off;                       // sentinel = total
                __syncwarp(gmask);
                uint32_t v = 0;
                for (uint32_t q0 = 0; q0 < total; q0 += SWEEP_U * GLANES) {
                    float4 p[SWEEP_U];
                    uint32_t ref[SWEEP_U];
#pragma unroll
                    for (int t = 0; t < SWEEP_U; ++t) {
                        const uint32_t q = q0 + t * GLANES + gl;
                        if (q < total) {
                            while (lo_[v + 1] <= q) ++v;
                            ref[t] = lb_[v] * (uint32_t)m.cap + (q - lo_[v]);
                            p[t] = __ldg(m.points + ref[t]);
                        }
                    }
#pragma unroll
                    for (int t = 0; t < SWEEP_U; ++t) if (q0 + t * GLANES + gl < total) consider(p[t], ref[t]);
                }
                __syncwarp(gmask);                                          // the list is rebuilt by the group's next point
            }
            const int w = group_argmin(gmask, best.d2, best.id);
            best.d2 = __shfl_sync(gmask, best.d2, w);
            best.id = __shfl_sync(gmask, best.id, w);
            best.ref = __shfl_sync(gmask, best.ref, w);
            const float rx = __shfl_sync(gmask, bx, w), ry = __shfl_sync(gmask, by, w), rz = __shfl_sync(gmask, bz, w);
            if (best.id == NO_ID) { have &= ~2u; continue; }
            if (best.ref != pref_seen) {
                // Sigma_r (lanes 0..5) and its flag (lane 6): one memory level, skipped if the neighbour is the old one
                if (have_scan_cov) {
                    if (gl < 6) cinr = __ldg(m.cov + (size_t)best.ref * 6 + gl);
                    if (gl == 6) cinr = (float)__ldg(m.cov_ok + best.ref);
                }
                // its voxel (a stored point: always valid), one coordinate per lane
                const float rmine = r3 == 0 ? rx : (r3 == 1 ? ry : rz);
                const int krm = (int)floorf(__fdiv_rn(rmine, m.voxel));
                __syncwarp(gmask);                                  // the reads of ps above are done
                if (gl < 3) { ps.kr[gl] = krm; ps.pr[gl] = rmine; }
                __syncwarp(gmask);
                pref = best.ref;
            }
            have |= 2u;
            if (best.d2 > tau2) continue;                           // adaptive-threshold gate
            // ---- A9: this group's correspondence -> its 29 terms ------------------------------------------------------
            const bool full = have_scan_cov && __shfl_sync(gmask, cinr, base + 6) != 0.f && __shfl_sync(gmask, cin, base + 6) != 0.f;
            const double px = (double)pfx, py = (double)pfy, pz = (double)pfz;
            const double d0 = (double)rx - px, d1 = (double)ry - py, d2 = (double)rz - pz;   // Eq. 3
            double M[6] = {1.0, 0.0, 0.0, 1.0, 0.0, 1.0};                // SA fallback: Sigma_r = I, Sigma_s = 0
            if (full) {
                // S = Sigma_r + R Sigma_s R^T (Eq. 4): lane e < 6 computes entry e = (i, j) of the upper triangle
                const int e = min(gl, 5);
                const int ei = e < 3 ? 0 : (e < 5 ? 1 : 2), ej = e < 3 ? e : (e < 5 ? e - 2 : 2);
                const double a = s_T.R[3 * ei], b = s_T.R[3 * ei + 1], c = s_T.R[3 * ei + 2];
                const float* cs = s_cs[slot];
                const double s0 = cs[0], s1 = cs[1], s2 = cs[2], s3 = cs[3], s4 = cs[4], s5 = cs[5];
                const double u0 = a * s0 + b * s1 + c * s2, u1 = a * s1 + b * s3 + c * s4, u2 = a * s2 + b * s4 + c * s5;
                const double cr_mine = (double)__shfl_sync(gmask, cinr, base + e);
                const double Sm = cr_mine + (u0 * s_T.R[3 * ej] + u1 * s_T.R[3 * ej + 1] + u2 * s_T.R[3 * ej + 2]);
                double S[6];
#pragma unroll
                for (int q = 0; q < 6; ++q) S[q] = shfl_d(gmask, Sm, base + q);
                double Mi[6];
                if (inv_sym3(S, Mi)) {
#pragma unroll
                    for (int q = 0; q < 6; ++q) M[q] = Mi[q];
                }
            }
            const double Md0 = M[0] * d0 + M[1] * d1 + M[2] * d2;
            const double Md1 = M[1] * d0 + M[3] * d1 + M[4] * d2;
            const double Md2 = M[2] * d0 + M[4] * d1 + M[5] * d2;
            const double e2 = d0 * Md0 + d1 * Md1 + d2 * Md2;
            const double wgt = robust_weight(P.kernel, e2, kappa);
            // the group's vector u: one or two entries per lane
            if (gl < 6) {
#pragma unroll
                for (int q = 0; q < 6; ++q) if (gl == q) u[q] = M[q];       // (no dynamic register indexing)
            } else if (gl == 6) { u[U_MD] = Md0; u[U_MD + 1] = Md1; u[U_MD + 2] = Md2; u[U_E2] = e2; }
            else { u[U_P] = px; u[U_P + 1] = py; u[U_P + 2] = pz; u[U_ZERO] = 0.0; u[U_ONE] = 1.0; }
            __syncwarp(gmask);
            auto term = [&](uint32_t en, bool store_x) -> double {
                const double val = u[en & 31u] * u[(en >> 5) & 31u] - u[(en >> 10) & 31u] * u[(en >> 15) & 31u];
                const uint32_t xs = en >> 22;
                if (store_x && xs) u[U_X + xs - 1] = val;
                const uint32_t ck = (en >> 20) & 3u;
                return (ck == COEF_W ? wgt : (ck == COEF_MW ? -wgt : 1.0)) * val;
            };
#pragma unroll
            for (int q = 0; q < TERM_SLOTS - 1; ++q) if (q * GLANES + gl < 24) acc[q] += term(enc[q], true);   // round 1
            __syncwarp(gmask);                                      // the nine X are in u
            if (gl < 8) acc[TERM_SLOTS - 1] += term(enc[TERM_SLOTS - 1], false);
            __syncwarp(gmask);                                      // u is rewritten by the group's next point
        }
        // ---- A10: lane-wise over the warp's 32 / GLANES groups, over the block's warps, then block row -> group of 16 blocks -> grid
        // as tagged words; every level summed in a fixed order
#pragma unroll
        for (int q = 0; q < TERM_SLOTS; ++q) {
            double v = acc[q];
#pragma unroll
            for (int d = GLANES; d < 32; d <<= 1) v += __shfl_xor_sync(FULL, v, d);
            const int col = q < TERM_SLOTS - 1 ? q * GLANES + lane : 24 + lane;
            if (q < TERM_SLOTS - 1 ? (lane < GLANES && col < 24) : lane < 8) s_part[wib][col] = v;
        }
        __syncthreads();
        if (wib == 0) {
            double t = 0.0;
#pragma unroll
            for (int w8 = 0; w8 < GWARPS; ++w8) t += s_part[w8][lane];
            put_tagged(P.scratch.rows + (size_t)blockIdx.x * TSTRIDE + c_term_store[lane], t, tag);
        }
        if (blockIdx.x % GROUP == 0) {   // group leader: fold the group's rows into one
            const int group = blockIdx.x / GROUP, n_groups = (G + GROUP - 1) / GROUP;
            const int group_rows = min(GROUP, G - group * GROUP);
            const double t = block_sum_tagged(P.scratch.rows, group * GROUP, group_rows, tag, lane, wib, s_red);
            if (n_groups > 1 && wib == 0) put_tagged(P.scratch.grows + (size_t)group * TSTRIDE + lane, t, tag);
            if (blockIdx.x == 0) {       // block 0: final sum (a single group: it has it already), solve, publish
                const double t2 = n_groups > 1 ? block_sum_tagged(P.scratch.grows, 0, n_groups, tag, lane, wib, s_red) : t;
                if (wib == 0) {
                    s_red[0][lane] = t2;
                    __syncwarp();
                    solve_and_publish(P, s_red[0], s_T, it, lane, tag);
                }
            }
        }
        // ---- grid-wide wait for the new pose: all blocks are co-resident (cooperative launch) -----------------------
        __syncthreads();                                      // the groups / the sums have finished reading s_T, s_part
        if (wib == 0) {
            // ONE lane per block polls the `done` word (written last); only when it carries this iteration's tag do the
            // other twelve lanes fetch their words (each still self-validating): the solver's stores do not queue behind
            // poll traffic in that L2 slice
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
    // sized for the capacity n; the kernel works with min(n, *d_n) points and the blocks it does not need leave at once
    int64_t grid = map->gicp_max_grid;
    const int64_t need = (n + 3) / 4;
    if (need < grid) grid = need;
    if (grid < 1) grid = 1;
    P.sm_count = map->sm_count;
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
