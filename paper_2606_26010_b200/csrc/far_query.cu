// far_query.cu -- 27-voxel nearest neighbour (A6) and k-nearest covariance (A7), one warp per query.
//
// PAPER.md:62 "the algorithm searches the voxel containing it as well as all surrounding ones (27 in total)",
// PAPER.md:80 "closest Euclidean neighbor" (k = 1), PAPER.md:68-76 (k = 10 -> Eq. 1).
//
// Warp-cooperative design: lanes 0..26 each probe one neighbour voxel (27 independent hash lookups in flight
// at once); the query's own voxel is swept first and bounds the search (far_common.cuh::warp_nearest), the
// counts of the voxels that can still matter are prefix-summed across the warp, and the warp sweeps that
// *flattened* candidate list 32 points at a time -- consecutive lanes read consecutive float4 of a bucket, so the
// gathers coalesce and no lane idles on a half-empty voxel.  Distances are FP64 with a fixed operation order (R6)
// so the arg-min is bit-identical to the definition; the arg-min itself is three redux.sync steps.
#include "far_internal.h"

using namespace far;

namespace far {

constexpr int QWARPS = 8;   // warps (= queries in flight) per block

// USE_OCC: the L2-resident occupancy bitmap is consulted before the table (far_common.cuh::find_voxel).  Chosen by the
// host when the table is more than twice the size of L2: on the 20 M-point map of C5 it lifts v = 0.25 / 0.5 from 1.27 / 1.24
// to 1.66 / 1.59 G queries/s (three quarters of the probes of absent voxels no longer reach DRAM); on tables that fit L2
// it is one more load per probe for nothing (C2 map: -3 %).
template <bool USE_OCC>
__global__ void __launch_bounds__(QWARPS * 32) nn_kernel(MapView m, const float* __restrict__ q, int64_t n, int stride,
                                                          uint32_t* __restrict__ out_id, float* __restrict__ out_d2) {
    __shared__ CandList s_list[QWARPS];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const int64_t nwarps = (int64_t)gridDim.x * QWARPS;
    for (int64_t i = (int64_t)blockIdx.x * QWARPS + wib; i < n; i += nwarps) {
        const float* qq = q + i * stride;
        const float qx = __ldg(qq), qy = __ldg(qq + 1), qz = __ldg(qq + 2);
        int k[3];
        uint32_t id = NO_ID;
        float d2 = __int_as_float(0x7F800000);
        if (voxel_index(qx, qy, qz, m.voxel, k)) {
            float rx, ry, rz;
            const Best b = warp_nearest<USE_OCC>(m, qx, qy, qz, k, lane, s_list[wib], rx, ry, rz);
            if (b.id != NO_ID) { id = b.id; d2 = __double2float_rn(b.d2); }
        }
        if (lane == 0) { out_id[i] = id; out_d2[i] = d2; }
        __syncwarp();
    }
}

__global__ void __launch_bounds__(QWARPS * 32) count27_kernel(MapView m, const float* __restrict__ q, int64_t n, int stride,
                                                               int32_t* __restrict__ out, int32_t* __restrict__ out_voxels) {
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const int64_t nwarps = (int64_t)gridDim.x * QWARPS;
    for (int64_t i = (int64_t)blockIdx.x * QWARPS + wib; i < n; i += nwarps) {
        const float* qq = q + i * stride;
        int k[3];
        uint32_t cnt = 0, bucket = NO_BUCKET;
        if (voxel_index(__ldg(qq), __ldg(qq + 1), __ldg(qq + 2), m.voxel, k)) probe27_regs(m, k, lane, cnt, bucket);
        const unsigned occ = __ballot_sync(FULL, cnt > 0);
        const int total = (int)__reduce_add_sync(FULL, cnt);
        if (lane == 0) {
            out[i] = total;
            if (out_voxels) out_voxels[i] = __popc(occ);
        }
    }
}

// ---- A7: k nearest by (d2, id) -> Eq. 1 -----------------------------------------------------------------------
// Two mappings of the same selection.
//  (a) Covariances of the points an insert accepted: ONE WARP PER TOUCHED VOXEL.  The accepted points of a
//      voxel are positions c0 .. c0 + n_new - 1 of its bucket and they all share the same 27-voxel candidate set, so the
//      warp probes the 27 neighbours once (27 lanes, one lookup each), stages every candidate point in shared memory with
//      coalesced loads that are all in flight together (north_star: "points staged in shared memory"), and then serves the
//      voxel's queries from there: G = 32 / pow2(n_new) lanes per query, each scanning a strided share of the staged list.
//      A lane keeps its KP = 12 best candidates as ONE 32-bit key each, in registers: the FP32 squared distance with its
//      11 low mantissa bits replaced by the candidate's index in the staged list, so unsigned order = distance order
//      (coarsened to 2^-12 relative) and inserting is a branch-free min/max chain; the G partial lists are merged with a
//      shuffle butterfly.  The exact FP64 (d2, id) selection of R6 then runs on those 12 only: the (count - k) largest are
//      dropped.  The result is PROVEN to be the definition's before it is used: a candidate that was not kept has a coarse
//      key >= the 12th kept one, hence an exact d2 >= W (1 - 3e-7) with W that key's distance bits; if the exact k-th
//      distance is below W (1 - 1e-6) no such candidate can precede it.  Otherwise (a near-tie across the 10th..12th
//      neighbour, ~1e-3 of the queries; always on lattice data; always when k > 10) the warp selects that query's k nearest
//      exactly, as k successive (d2, id) minima over the staged list.
//      Round-2 profile of the previous mapping (one thread per query: 1,414 warps for a C2 frame, 8 per SM, every lane
//      walking ~230 candidates behind 27 dependent lookups): 92 us, 41 % long-scoreboard stalls at 12.7 % warps active.
//  (b) A free-standing query (far_map_knn_cov: a downsampled scan point against the scan-local map; one query per
//      voxel, nothing to share): one WARP per query, lane l keeps the k smallest of its candidates as a sorted column,
//      then k rounds of warp arg-min over the column heads.
struct __align__(16) Cand {
    double d2;
    uint32_t id;
    uint32_t idx;      // reference bucket * cap + position of the candidate
};

__device__ __forceinline__ bool cand_less(double d2, uint32_t id, const Cand& c) {
    return d2 < c.d2 || (d2 == c.d2 && id < c.id);
}

// Eq. 1: C = Sigma_hat + eps I ; Sigma = (C^-1 / ||C^-1||_F)^-1 = ||C^-1||_F C.  FP64 throughout.
__device__ __forceinline__ bool regularised_cov(const double sc[6], double eps, float out[6]) {
    const double a0 = sc[0] + eps, a1 = sc[1], a2 = sc[2], a4 = sc[3] + eps, a5 = sc[4], a8 = sc[5] + eps;
    // symmetric: a3 = a1, a6 = a2, a7 = a5
    const double c00 = a4 * a8 - a5 * a5;
    const double c01 = a5 * a2 - a1 * a8;
    const double c02 = a1 * a5 - a4 * a2;
    const double det = a0 * c00 + a1 * c01 + a2 * c02;
    if (!(det != 0.0) || !isfinite(det)) return false;
    // ||C^-1||_F = ||adj(C)||_F / |det|
    const double c11 = a0 * a8 - a2 * a2, c12 = a2 * a1 - a0 * a5, c22 = a0 * a4 - a1 * a1;
    const double fro = sqrt(c00 * c00 + c11 * c11 + c22 * c22 + 2.0 * (c01 * c01 + c02 * c02 + c12 * c12)) / fabs(det);
    out[0] = (float)(fro * a0); out[1] = (float)(fro * a1); out[2] = (float)(fro * a2);
    out[3] = (float)(fro * a4); out[4] = (float)(fro * a5); out[5] = (float)(fro * a8);
    return true;
}

constexpr int KP = 12;              // candidates a lane keeps (coarse keys)
constexpr int STAGE_U = 4;          // staging loads in flight per lane

// per-warp shared memory of mapping (a): the staged candidates, the list bookkeeping, the indices an exact selection picks
__host__ __device__ inline size_t cov_task_bytes(int cap) {
    return (size_t)27 * cap * sizeof(float4) + ((sizeof(CandList) + 15) & ~(size_t)15) + 64 * sizeof(int);
}

// R7 for the staged candidates named by sel[0 .. kk): mean and centred second moments in that order (1/k), then Eq. 1
__device__ __forceinline__ bool cov_of_selection(const MapView& m, const float4* cand, const int* sel, float out[6]) {
    const int kk = m.k_cov;
    const double inv_k = 1.0 / (double)kk;
    double mx = 0.0, my = 0.0, mz = 0.0;
    for (int r = 0; r < kk; ++r) { const float4 p = cand[sel[r]]; mx += (double)p.x; my += (double)p.y; mz += (double)p.z; }
    mx *= inv_k; my *= inv_k; mz *= inv_k;
    double sc[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    for (int r = 0; r < kk; ++r) {
        const float4 p = cand[sel[r]];
        const double dx = (double)p.x - mx, dy = (double)p.y - my, dz = (double)p.z - mz;
        sc[0] += dx * dx; sc[1] += dx * dy; sc[2] += dx * dz; sc[3] += dy * dy; sc[4] += dy * dz; sc[5] += dz * dz;
    }
#pragma unroll
    for (int a = 0; a < 6; ++a) sc[a] *= inv_k;
    return regularised_cov(sc, m.cov_eps, out);
}

// exact selection for ONE query by the whole warp: k successive minima of (d2, id) over the staged list (R6 order); the
// chosen indices land in sel[], lane 0 computes Eq. 1.  total >= k.  All 32 lanes must call.
__device__ __noinline__ bool warp_cov_exact(const MapView& m, const float4* cand, int total, float qx, float qy, float qz, int lane, int* sel,
                                            float out[6]) {
    const int kk = m.k_cov;
    const double INF = __longlong_as_double(0x7FF0000000000000ll);
    double ld = -1.0;                    // last chosen (d2, id): every d2 >= 0 follows it
    uint32_t lid = 0;
    for (int r = 0; r < kk; ++r) {
        double bd = INF;
        uint32_t bid = NO_ID;
        int bj = 0;
        for (int j = lane; j < total; j += 32) {
            const float4 p = cand[j];
            const double d2 = dist2(qx, qy, qz, p.x, p.y, p.z);
            const uint32_t id = __float_as_uint(p.w);
            const bool after = d2 > ld || (d2 == ld && id > lid);
            if (after && (d2 < bd || (d2 == bd && id < bid))) { bd = d2; bid = id; bj = j; }
        }
        const int w = warp_argmin(bd, bid);
        ld = __shfl_sync(FULL, bd, w);
        lid = __shfl_sync(FULL, bid, w);
        if (lane == w) sel[r] = bj;
    }
    __syncwarp();
    bool ok = false;
    if (lane == 0) ok = cov_of_selection(m, cand, sel, out);
    __syncwarp();
    return ok;                            // valid in lane 0
}

// mapping (a): the covariances of stored points c0 .. c0 + n_new - 1 of bucket b, by one warp (all 32 lanes must call)
// neighbour l of the near-first order: l = 0 the voxel itself, 1..6 face, 7..18 edge, 19..26 corner neighbours;
// packed as (dx + 1) | (dy + 1) << 2 | (dz + 1) << 4
__constant__ uint8_t c_near_first[27] = {
    0x15,
    0x14, 0x16, 0x11, 0x19, 0x05, 0x25,
    0x10, 0x12, 0x18, 0x1A, 0x04, 0x06, 0x24, 0x26, 0x01, 0x09, 0x21, 0x29,
    0x00, 0x02, 0x08, 0x0A, 0x20, 0x22, 0x28, 0x2A};

__device__ __forceinline__ void warp_cov_task(const MapView& m, unsigned long long vkey, uint32_t b, uint32_t c0, uint32_t n_new, int lane,
                                              float4* cand, CandList& L, int* sel) {
    const int cap = m.cap, kk = m.k_cov;
    const size_t first = (size_t)b * cap + c0;
    auto write_out = [&](uint32_t q, bool ok, const float c[6]) {
        float* o = m.cov + (first + q) * 6;
        o[0] = ok ? c[0] : 1.f; o[1] = ok ? c[1] : 0.f; o[2] = ok ? c[2] : 0.f; o[3] = ok ? c[3] : 1.f; o[4] = ok ? c[4] : 0.f; o[5] = ok ? c[5] : 1.f;
        m.cov_ok[first + q] = ok ? 1 : 0;
    };
    // the 27 lookups in NEAR-FIRST order (lane 0 the voxel itself, then face, edge, corner neighbours): the staged list
    // starts with the voxel's own points and a query's 12th-best distance is tight before the far voxels come up
    int k[3];
    unpack_key(vkey, k);
    uint32_t cnt = 0, bucket = NO_BUCKET;
    int nbr = 0;
    if (lane < 27) {
        nbr = c_near_first[lane];
        const int nx = k[0] + (nbr & 3) - 1, ny = k[1] + ((nbr >> 2) & 3) - 1, nz = k[2] + ((nbr >> 4) & 3) - 1;
        if (index_in_range(nx) && index_in_range(ny) && index_in_range(nz)) bucket = find_voxel(m, pack_key(nx, ny, nz), cnt);
    }
    const unsigned occ = __ballot_sync(FULL, cnt > 0);
    const int total = cand_build(L, cnt, bucket, lane);
    int* nb = sel + 32;                  // offset code of compact voxel c
    if (cnt > 0) nb[__popc(occ & ((1u << lane) - 1u))] = nbr;
    const int nvox = __popc(occ);
    if (total < kk) {                    // fewer than k candidates in the 27 voxels: every query of the voxel is invalid
        const float none[6] = {1.f, 0.f, 0.f, 1.f, 0.f, 1.f};
        for (uint32_t q = lane; q < n_new; q += 32) write_out(q, false, none);
        __syncwarp();
        return;
    }
    // stage every candidate (x, y, z, id bits): STAGE_U x 32 independent loads in flight
    {
        CandIter ci;
        ci.before = 0;
        for (int j0 = 0, step = 0; j0 < total; j0 += 32 * STAGE_U) {
            float4 p[STAGE_U];
#pragma unroll
            for (int u = 0; u < STAGE_U; ++u) {
                const int j = j0 + 32 * u + lane;
                if (j0 + 32 * u < total) {                       // warp-uniform: cand_next wants every step, in order
                    const uint32_t ref = cand_next(L, ci, step, j, lane, cap);
                    ++step;
                    if (j < total) p[u] = __ldg(m.points + ref);
                }
            }
#pragma unroll
            for (int u = 0; u < STAGE_U; ++u) {
                const int j = j0 + 32 * u + lane;
                if (j < total) cand[j] = p[u];
            }
        }
    }
    __syncwarp();
    const int own = (int)c0;                                               // staged index of the voxel's first new point (its voxel is compact voxel 0)
    for (uint32_t q0 = 0; q0 < n_new; q0 += 32) {
        const uint32_t nq = min(32u, n_new - q0);
        int G = 1;                                                     // lanes per query: the largest power of two that fits
        while (2 * G * nq <= 32) G *= 2;
        const uint32_t qi = lane / G;
        const int sub = lane % G;
        const bool act = qi < nq;
        float qx = 0.f, qy = 0.f, qz = 0.f;
        if (act) { const float4 qp = cand[own + q0 + qi]; qx = qp.x; qy = qp.y; qz = qp.z; }
        bool need_exact = act && sub == 0 && kk > KP - 2;
        if (kk <= KP - 2) {
            // coarse keys of this lane's share of the list, sorted ascending in registers
            uint32_t key[KP];
#pragma unroll
            for (int i = 0; i < KP; ++i) key[i] = 0xFFFFFFFFu;
            if (act) {
                // squared FP32 gaps from the query to the six faces of its voxel, pulled in by 2^-19 |k| v (key rounding and
                // the FP32 arithmetic here): a neighbour voxel's distance lower bound is a sum of up to three of them
                float glo[3], ghi[3];
                const float qq[3] = {qx, qy, qz};
#pragma unroll
                for (int a = 0; a < 3; ++a) {
                    const float mg = (float)(abs(k[a]) + 2) * m.voxel * 1.9073486328125e-06f;
                    const float lo = fmaxf(qq[a] - (float)k[a] * m.voxel - mg, 0.f), hi = fmaxf((float)(k[a] + 1) * m.voxel - qq[a] - mg, 0.f);
                    glo[a] = lo * lo; ghi[a] = hi * hi;
                }
                for (int c = 0; c < nvox; ++c) {
                    const int j0 = L.off[c], j1 = c + 1 < nvox ? L.off[c + 1] : total;
                    if (c > 0 && key[KP - 1] != 0xFFFFFFFFu) {
                        // skip the voxel if even its nearest possible point cannot enter this lane's list: every candidate
                        // in it then has a coarse key above key[KP - 1] (0.2 % slack covers the key's 2^-12 coarsening)
                        const int o = nb[c];
                        const int ox = (o & 3) - 1, oy = ((o >> 2) & 3) - 1, oz = ((o >> 4) & 3) - 1;
                        const float lb = (ox < 0 ? glo[0] : (ox > 0 ? ghi[0] : 0.f)) + (oy < 0 ? glo[1] : (oy > 0 ? ghi[1] : 0.f)) +
                                         (oz < 0 ? glo[2] : (oz > 0 ? ghi[2] : 0.f));
                        if (lb * 0.998f > __uint_as_float(key[KP - 1] | 0x7FFu)) continue;
                    }
                    for (int j = j0 + sub; j < j1; j += G) {
                        const float4 p = cand[j];
                        const float fx = qx - p.x, fy = qy - p.y, fz = qz - p.z;
                        uint32_t x = (__float_as_uint(fmaf(fz, fz, fmaf(fy, fy, fx * fx))) & 0xFFFFF800u) | (uint32_t)j;
                        if (x < key[KP - 1]) {
#pragma unroll
                            for (int i = 0; i < KP; ++i) { const uint32_t lo = min(key[i], x); x = max(key[i], x); key[i] = lo; }
                        }
                    }
                }
            }
            // merge the G partial lists (disjoint shares): after the butterfly every lane of a group holds the group's best KP.
            // Two ascending lists a, b of KP keys: c[i] = min(a[i], b[KP-1-i]) are the KP smallest of the union, as a sequence
            // that rises and then falls; padded with four zeros at the end it is bitonic as a cycle, and one bitonic merge
            // network over 16 (the zeros are compile-time constants: their exchanges fold away) sorts it -- about 70
            // instructions a level, where inserting the partner's keys one by one through the min/max chain took ~190
            for (int d = 1; d < G; d <<= 1) {
                uint32_t c[16];
#pragma unroll
                for (int i = 0; i < KP; ++i) c[i] = min(key[i], __shfl_xor_sync(FULL, key[KP - 1 - i], d));
#pragma unroll
                for (int i = KP; i < 16; ++i) c[i] = 0u;
#pragma unroll
                for (int stride = 8; stride > 0; stride >>= 1) {
#pragma unroll
                    for (int i = 0; i < 16; ++i) {
                        if ((i & stride) == 0) {
                            const uint32_t lo = min(c[i], c[i + stride]), hi = max(c[i], c[i + stride]);
                            c[i] = lo; c[i + stride] = hi;
                        }
                    }
                }
#pragma unroll
                for (int i = 0; i < KP; ++i) key[i] = c[i + 16 - KP];       // the zeros sort to the front
            }
            if (act && sub == 0) {
                // exact (d2, id) of the kept candidates (R6); drop the (count - k) largest; prove; Eq. 1
                double d2e[KP];
                uint32_t ide[KP];
                int n_kept = 0;
#pragma unroll
                for (int i = 0; i < KP; ++i) {
                    d2e[i] = -1.0; ide[i] = 0;
                    if (key[i] != 0xFFFFFFFFu) {
                        const float4 p = cand[key[i] & 0x7FFu];
                        d2e[i] = dist2(qx, qy, qz, p.x, p.y, p.z);
                        ide[i] = __float_as_uint(p.w);
                        ++n_kept;
                    }
                }
                unsigned out_mask = 0;                                  // dropped or absent
#pragma unroll
                for (int i = 0; i < KP; ++i) if (key[i] == 0xFFFFFFFFu) out_mask |= 1u << i;
                for (int r = n_kept; r > kk; --r) {
                    double wd = -1.0;
                    uint32_t wid = 0;
                    int wi = 0;
#pragma unroll
                    for (int i = 0; i < KP; ++i) {
                        if (!(out_mask & (1u << i)) && (d2e[i] > wd || (d2e[i] == wd && ide[i] > wid))) { wd = d2e[i]; wid = ide[i]; wi = i; }
                    }
                    out_mask |= 1u << wi;
                }
                double kth = -1.0;                                      // exact k-th smallest distance
#pragma unroll
                for (int i = 0; i < KP; ++i) if (!(out_mask & (1u << i))) kth = fmax(kth, d2e[i]);
                bool proven = true;                                     // fewer than KP candidates in all: nothing was ever rejected
                if (key[KP - 1] != 0xFFFFFFFFu) proven = kth < (double)__uint_as_float(key[KP - 1] & 0xFFFFF800u) * (1.0 - 1e-6);
                if (!proven) {
                    need_exact = true;
                } else {
                    // mean and centred moments over the k chosen, in key order (fixed), 1/k; Eq. 1
                    const double inv_k = 1.0 / (double)kk;
                    double mx = 0.0, my = 0.0, mz = 0.0;
#pragma unroll
                    for (int i = 0; i < KP; ++i) {
                        if (!(out_mask & (1u << i))) { const float4 p = cand[key[i] & 0x7FFu]; mx += (double)p.x; my += (double)p.y; mz += (double)p.z; }
                    }
                    mx *= inv_k; my *= inv_k; mz *= inv_k;
                    double sc[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
#pragma unroll
                    for (int i = 0; i < KP; ++i) {
                        if (!(out_mask & (1u << i))) {
                            const float4 p = cand[key[i] & 0x7FFu];
                            const double dx = (double)p.x - mx, dy = (double)p.y - my, dz = (double)p.z - mz;
                            sc[0] += dx * dx; sc[1] += dx * dy; sc[2] += dx * dz; sc[3] += dy * dy; sc[4] += dy * dz; sc[5] += dz * dz;
                        }
                    }
#pragma unroll
                    for (int a = 0; a < 6; ++a) sc[a] *= inv_k;
                    float c[6];
                    const bool ok = regularised_cov(sc, m.cov_eps, c);
                    write_out(q0 + qi, ok, c);
                }
            }
        }
        // the queries the coarse keys could not settle: exact selection, one query at a time by the whole warp
        unsigned todo = __ballot_sync(FULL, need_exact);
        while (todo) {
            const int src = __ffs(todo) - 1;
            todo &= todo - 1;
            const float ex = __shfl_sync(FULL, qx, src), ey = __shfl_sync(FULL, qy, src), ez = __shfl_sync(FULL, qz, src);
            const uint32_t eq = __shfl_sync(FULL, q0 + qi, src);
            float c[6];
            const bool ok = warp_cov_exact(m, cand, total, ex, ey, ez, lane, sel, c);
            if (lane == 0) write_out(eq, ok, c);
        }
        __syncwarp();
    }
}

// tasks = the voxels an insert call added points to, queued by its commit kernel: {key lo, key hi, bucket, c0 | n_new << 8}.
// Two sweeps over the queue, the voxels with many new points first: they are the long jobs (a query gets 32 / pow2(n_new)
// lanes), and a warp that picks one up last would finish long after the others.
__global__ void __launch_bounds__(256, 3) knn_cov_refs_kernel(MapView m, const uint4* __restrict__ tasks, const unsigned int* __restrict__ d_n,
                                    int warps_per_block) {
    extern __shared__ __align__(16) char smem[];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    char* wbase = smem + (size_t)wib * cov_task_bytes(m.cap);
    float4* cand = reinterpret_cast<float4*>(wbase);
    CandList& L = *reinterpret_cast<CandList*>(wbase + (size_t)27 * m.cap * sizeof(float4));
    int* sel = reinterpret_cast<int*>(wbase + (size_t)27 * m.cap * sizeof(float4) + ((sizeof(CandList) + 15) & ~(size_t)15));
    const int64_t n = *d_n;
    const int64_t nwarps = (int64_t)gridDim.x * warps_per_block;
    for (int sweep = 0; sweep < 2; ++sweep) {
        for (int64_t t = (int64_t)blockIdx.x * warps_per_block + wib; t < n; t += nwarps) {
            const uint4 task = tasks[t];
            const uint32_t c0 = task.w & 0xFFu, n_new = task.w >> 8;
            if ((n_new > 8) == (sweep == 0))
                warp_cov_task(m, ((unsigned long long)task.y << 32) | task.x, task.z, c0, n_new, lane, cand, L, sel);
        }
    }
}

// same for calls larger than the task list: every stored point with id >= the call's first id is a new point.  A warp
// takes 32 table slots and serves the voxels among them that hold new points one after the other.
__global__ void __launch_bounds__(256) knn_cov_new_ids_kernel(MapView m, int warps_per_block) {
    extern __shared__ __align__(16) char smem[];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    char* wbase = smem + (size_t)wib * cov_task_bytes(m.cap);
    float4* cand = reinterpret_cast<float4*>(wbase);
    CandList& L = *reinterpret_cast<CandList*>(wbase + (size_t)27 * m.cap * sizeof(float4));
    int* sel = reinterpret_cast<int*>(wbase + (size_t)27 * m.cap * sizeof(float4) + ((sizeof(CandList) + 15) & ~(size_t)15));
    const uint32_t first_id = (uint32_t)m.ctr->call_first_id;
    const int64_t nwarps = (int64_t)gridDim.x * warps_per_block;
    for (int64_t s0 = ((int64_t)blockIdx.x * warps_per_block + wib) * 32; s0 < m.slots; s0 += nwarps * 32) {
        Entry e;
        e.key = KEY_EMPTY; e.bucket = NO_BUCKET; e.cr = 0;
        if (s0 + lane < m.slots) e = m.table[s0 + lane];
        uint32_t cnt = entry_count(e.cr), c0 = cnt;
        if (e.key == KEY_EMPTY || e.bucket >= BUCKET_PENDING) cnt = c0 = 0;
        while (c0 > 0 && m.ids[(size_t)e.bucket * m.cap + c0 - 1] >= first_id) --c0;     // ids ascend: the new points are a suffix
        unsigned todo = __ballot_sync(FULL, cnt > c0);
        while (todo) {
            const int src = __ffs(todo) - 1;
            todo &= todo - 1;
            const uint32_t b = __shfl_sync(FULL, e.bucket, src), f = __shfl_sync(FULL, c0, src), c = __shfl_sync(FULL, cnt, src);
            const uint32_t klo = __shfl_sync(FULL, (uint32_t)e.key, src), khi = __shfl_sync(FULL, (uint32_t)(e.key >> 32), src);
            warp_cov_task(m, ((unsigned long long)khi << 32) | klo, b, f, c - f, lane, cand, L, sel);
        }
    }
}

// (b) one warp = one free-standing query: 27 lookups by 27 lanes, flattened list, per-lane sorted columns, k rounds of
// warp arg-min, Eq. 1 by lanes 0..8
__device__ __forceinline__ bool warp_knn_cov(const MapView& m, float qx, float qy, float qz, int lane, Cand* col, double* mom,
                                             CandList& L, float cov[6]) {
    const int cap = m.cap, kk = m.k_cov;
    cov[0] = 1.f; cov[1] = 0.f; cov[2] = 0.f; cov[3] = 1.f; cov[4] = 0.f; cov[5] = 1.f;
    int k[3];
    if (!voxel_index(qx, qy, qz, m.voxel, k)) return false;
    uint32_t pcnt, pbucket;
    probe27_regs(m, k, lane, pcnt, pbucket);
    const int total = cand_build(L, pcnt, pbucket, lane);
    if (total < kk) { __syncwarp(); return false; }
    const double INF = __longlong_as_double(0x7FF0000000000000ll);
    int cnt = 0;
    CandIter ci;
    ci.before = 0;
    for (int j = lane, step = 0; j < total; j += 32, ++step) {
        const uint32_t ref = cand_next(L, ci, step, j, lane, cap);
        const float4 p = __ldg(m.points + ref);
        const double d2 = dist2(qx, qy, qz, p.x, p.y, p.z);   // R6
        const uint32_t id = __float_as_uint(p.w);
        int q = cnt;
        if (cnt == kk) {
            if (!cand_less(d2, id, col[(kk - 1) * 32 + lane])) continue;    // cannot enter this lane's top k
            q = kk - 1;
        } else {
            ++cnt;
        }
        while (q > 0) {
            const Cand c = col[(q - 1) * 32 + lane];
            if (!cand_less(d2, id, c)) break;
            col[q * 32 + lane] = c;
            --q;
        }
        Cand e;
        e.d2 = d2; e.id = id; e.idx = ref;
        col[q * 32 + lane] = e;
    }
    // k rounds of warp arg-min over the column heads
    int h = 0;
    Cand head;
    head.d2 = INF; head.id = NO_ID; head.idx = 0;
    if (cnt > 0) head = col[lane];
    uint32_t myref = 0;
    for (int r = 0; r < kk; ++r) {
        const int w = warp_argmin(head.d2, head.id);
        const uint32_t wref = __shfl_sync(FULL, head.idx, w);
        if (lane == r) myref = wref;
        if (lane == w) {
            ++h;
            if (h < cnt) head = col[h * 32 + lane];
            else { head.d2 = INF; head.id = NO_ID; }
        }
    }
    // lane r < k holds the r-th neighbour: positions through shared memory, then lane a < 3 sums coordinate a in neighbour
    // order (R7: 1/k) and lane a < 6 accumulates centred product a, also in order
    __syncwarp();
    double* nb = mom;                                         // [k][3] positions, then [3] mean, then [6] moments
    if (lane < kk) {
        const float4 p = __ldg(m.points + myref);
        nb[3 * lane] = (double)p.x; nb[3 * lane + 1] = (double)p.y; nb[3 * lane + 2] = (double)p.z;
    }
    __syncwarp();
    const double inv_k = 1.0 / (double)kk;
    double* mean = nb + 3 * kk;
    double* mo = mean + 3;
    if (lane < 3) {
        double sacc = 0.0;
        for (int r = 0; r < kk; ++r) sacc += nb[3 * r + lane];
        mean[lane] = sacc * inv_k;
    }
    __syncwarp();
    if (lane < 6) {
        // (xx,xy,xz,yy,yz,zz) -> axis pair (i,j)
        const int i = lane < 3 ? 0 : (lane < 5 ? 1 : 2);
        const int j = lane < 3 ? lane : (lane < 5 ? lane - 2 : 2);
        const double mi = mean[i], mj = mean[j];
        double sacc = 0.0;
        for (int r = 0; r < kk; ++r) sacc += (nb[3 * r + i] - mi) * (nb[3 * r + j] - mj);
        mo[lane] = sacc * inv_k;
    }
    __syncwarp();
    double sc[6];
#pragma unroll
    for (int a = 0; a < 6; ++a) sc[a] = mo[a];
    __syncwarp();
    float out[6];
    if (!regularised_cov(sc, m.cov_eps, out)) return false;
#pragma unroll
    for (int a = 0; a < 6; ++a) cov[a] = out[a];
    return true;
}

// per-warp shared memory of mapping (b).  The candidate list comes last, only as many of its step masks as this cap
// needs are allocated, and the moments of Eq. 1 later take its place: at k = 10, cap 20 a warp then takes 5.4 KB, five 8-warp blocks fit an SM, and the 5,352 queries of
// a C2 frame run as ONE wave of 5,920 warps (at 5.9 KB it was four blocks: 4,736 warps and a second wave for the rest)
__host__ __device__ inline size_t knn_warp_bytes(int k, int cap) {
    const size_t mask_words = ((size_t)27 * cap + 31) / 32;
    const size_t list = sizeof(CandList) - (CAND_STEPS - mask_words) * sizeof(uint32_t), mom = (size_t)(3 * k + 9) * sizeof(double);
    return (size_t)32 * k * sizeof(Cand) + (list > mom ? list : mom);      // the moments reuse the list's place: it has served by then
}

// queries given as points (far_map_knn_cov); n read from the device if d_n != nullptr
__global__ void __launch_bounds__(256, 5) knn_cov_points_kernel(MapView m, const float* __restrict__ q, int64_t n, const int64_t* __restrict__ d_n,
                                      int stride, float* __restrict__ cov6, uint8_t* __restrict__ valid, int warps_per_block) {
    extern __shared__ __align__(16) char smem[];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    char* wbase = smem + (size_t)wib * ((knn_warp_bytes(m.k_cov, m.cap) + 15) & ~(size_t)15);
    Cand* col = reinterpret_cast<Cand*>(wbase);
    double* mom = reinterpret_cast<double*>(wbase + (size_t)32 * m.k_cov * sizeof(Cand));
    CandList& L = *reinterpret_cast<CandList*>(wbase + (size_t)32 * m.k_cov * sizeof(Cand));
    if (d_n) n = min(n, *d_n);
    const int64_t nwarps = (int64_t)gridDim.x * warps_per_block;
    for (int64_t i = (int64_t)blockIdx.x * warps_per_block + wib; i < n; i += nwarps) {
        const float* qq = q + i * stride;
        float c[6];
        const bool ok = warp_knn_cov(m, __ldg(qq), __ldg(qq + 1), __ldg(qq + 2), lane, col, mom, L, c);
        if (lane < 6) cov6[i * 6 + lane] = c[lane];
        if (lane == 0) valid[i] = ok ? 1 : 0;
    }
}

struct KnnLaunch { int warps, grid; size_t smem; };

// The shared-memory opt-in and the occupancy query are slow host calls: done once per (kernel, bytes per warp, device) and
// cached (the frame chain launches two of these kernels per scan).
template <class K>
static int knn_launch_cfg(const far_map* map, K kernel, size_t per_warp, int64_t work_warps, KnnLaunch& L) {
    struct Cached { size_t per_warp; int dev; int warps, per_sm; size_t smem; };
    static Cached cache[16] = {};             // one table per kernel instantiation
    static int n_cached = 0;
    static size_t attr_bytes[8] = {};         // largest dynamic shared-memory opt-in made for this kernel, per device
    per_warp = (per_warp + 15) & ~(size_t)15;
    const int dev = map->device;
    Cached fresh;
    Cached* hit = nullptr;
    for (int q = 0; q < n_cached; ++q) if (cache[q].per_warp == per_warp && cache[q].dev == dev) hit = &cache[q];
    if (!hit) {
        int warps = (int)(100 * 1024 / per_warp);
        if (warps > 8) warps = 8;
        if (warps < 1) warps = 1;
        fresh.per_warp = per_warp; fresh.dev = dev; fresh.warps = warps; fresh.smem = per_warp * warps; fresh.per_sm = 0;
    }
    Cached& c = hit ? *hit : fresh;
    if (c.smem > attr_bytes[dev & 7] || dev >= 8) {   // the opt-in is per function: only ever raise it
        FAR_CUDA(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c.smem));
        attr_bytes[dev & 7] = c.smem;
    }
    if (!hit) {
        int per_sm = 0;
        FAR_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, c.warps * 32, c.smem));
        c.per_sm = per_sm < 1 ? 1 : per_sm;
        if (n_cached < 16) cache[n_cached++] = c;
    }
    L.warps = c.warps; L.smem = c.smem;
    int64_t grid = (int64_t)map->sm_count * c.per_sm;
    const int64_t need = (work_warps + c.warps - 1) / c.warps;
    if (need < grid) grid = need;
    if (grid < 1) grid = 1;
    L.grid = (int)grid;
    return FAR_OK;
}

int launch_knn_cov_refs(const far_map* map, const uint32_t* d_tasks, const unsigned int* d_n, int64_t n_max, cudaStream_t st) {
    KnnLaunch L;
    int rc = knn_launch_cfg(map, knn_cov_refs_kernel, cov_task_bytes(map->view.cap), n_max, L);
    if (rc != FAR_OK) return rc;
    FAR_LAUNCH(knn_cov_refs_kernel, L.grid, L.warps * 32, L.smem, st, map->view, reinterpret_cast<const uint4*>(d_tasks), d_n, L.warps);
    FAR_CUDA(cudaGetLastError());
    return FAR_OK;
}

int launch_knn_cov_new_ids(const far_map* map, cudaStream_t st) {
    KnnLaunch L;
    int rc = knn_launch_cfg(map, knn_cov_new_ids_kernel, cov_task_bytes(map->view.cap), (map->view.slots + 31) / 32, L);
    if (rc != FAR_OK) return rc;
    FAR_LAUNCH(knn_cov_new_ids_kernel, L.grid, L.warps * 32, L.smem, st, map->view, L.warps);
    FAR_CUDA(cudaGetLastError());
    return FAR_OK;
}

}  // namespace far

extern "C" {

int far_map_nn(const far_map_t* map, const float* d_q, int64_t m, int stride, uint32_t* d_id, float* d_d2, void* stream) {
    if (!map || m < 0 || (stride != 3 && stride != 4) || (m > 0 && (!d_q || !d_id || !d_d2))) return FAR_ERR_ARG;
    if (m == 0) return FAR_OK;
    // exactly one resident wave (the kernel is a grid-stride loop): a grid larger than the residency the register
    // count allows leaves a partial second wave behind
    static int per_sm = 0;
    if (per_sm == 0) {
        int v = 0, w = 0;
        FAR_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&v, nn_kernel<false>, QWARPS * 32, 0));
        FAR_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&w, nn_kernel<true>, QWARPS * 32, 0));
        v = v < w ? v : w;
        per_sm = v < 1 ? 1 : v;
    }
    int64_t grid = (int64_t)map->sm_count * per_sm;
    const int64_t need = (m + QWARPS - 1) / QWARPS;
    if (need < grid) grid = need;
    const bool use_occ = (size_t)map->view.slots * sizeof(Entry) > 2 * (size_t)map->l2_bytes;
    {
        far::LaunchScope ls_("nn_kernel", (cudaStream_t)stream);
        if (use_occ) nn_kernel<true><<<(int)grid, QWARPS * 32, 0, (cudaStream_t)stream>>>(map->view, d_q, m, stride, d_id, d_d2);
        else nn_kernel<false><<<(int)grid, QWARPS * 32, 0, (cudaStream_t)stream>>>(map->view, d_q, m, stride, d_id, d_d2);
    }
    FAR_CUDA(cudaGetLastError());
    return FAR_OK;
}

int far_map_count27(const far_map_t* map, const float* d_q, int64_t m, int stride, int32_t* d_count, int32_t* d_voxels,
                    void* stream) {
    if (!map || m < 0 || (stride != 3 && stride != 4) || (m > 0 && (!d_q || !d_count))) return FAR_ERR_ARG;
    if (m == 0) return FAR_OK;
    int64_t grid = (int64_t)map->sm_count * 8;
    const int64_t need = (m + QWARPS - 1) / QWARPS;
    if (need < grid) grid = need;
    FAR_LAUNCH(count27_kernel, (int)grid, QWARPS * 32, 0, (cudaStream_t)stream, map->view, d_q, m, stride, d_count, d_voxels);
    FAR_CUDA(cudaGetLastError());
    return FAR_OK;
}

static int knn_cov_impl(const far_map_t* map, const float* d_q, int64_t m, const int64_t* d_m, int stride, float* d_cov6,
                        uint8_t* d_valid, void* stream) {
    if (!map || m < 0 || (stride != 3 && stride != 4) || (m > 0 && (!d_q || !d_cov6 || !d_valid))) return FAR_ERR_ARG;
    if (m == 0) return FAR_OK;
    KnnLaunch L;
    int rc = knn_launch_cfg(map, knn_cov_points_kernel, knn_warp_bytes(map->view.k_cov, map->view.cap), m, L);
    if (rc != FAR_OK) return rc;
    FAR_LAUNCH(knn_cov_points_kernel, L.grid, L.warps * 32, L.smem, (cudaStream_t)stream, map->view, d_q, m, d_m, stride, d_cov6,
                                                                                  d_valid, L.warps);
    FAR_CUDA(cudaGetLastError());
    return FAR_OK;
}

int far_map_knn_cov(const far_map_t* map, const float* d_q, int64_t m, int stride, float* d_cov6, uint8_t* d_valid,
                    void* stream) {
    return knn_cov_impl(map, d_q, m, nullptr, stride, d_cov6, d_valid, stream);
}

int far_map_knn_cov_dev(const far_map_t* map, const float* d_q, const int64_t* d_m, int64_t m_max, int stride,
                        float* d_cov6, uint8_t* d_valid, void* stream) {
    if (!d_m) return FAR_ERR_ARG;
    return knn_cov_impl(map, d_q, m_max, d_m, stride, d_cov6, d_valid, stream);
}

}  // extern "C"
