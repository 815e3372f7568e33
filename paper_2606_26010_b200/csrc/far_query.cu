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
            const Best b = warp_nearest(m, qx, qy, qz, k, lane, s_list[wib], rx, ry, rz);
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
//  (a) Covariances of the points an insert accepted: ONE THREAD PER QUERY.  The accepted points arrive
//      grouped by voxel, so consecutive lanes of a warp are (mostly) points of the same voxel: they walk the same 27
//      voxels, their loads of table entries and candidate points coalesce into a few sectors served by L1, and they
//      run in lockstep.  A lane walks its 27 voxels in NEAR-FIRST order (own voxel, 6 face, 12 edge, 8 corner
//      neighbours) so that its k-th best is tight after the first voxel, tests every candidate in FP32 against that
//      bound (relative error of the FP32 d2 < 3e-7, margin 1e-6) and only appends the survivors to a short list; the
//      exact FP64 distance of R6 and the sorted insertion run over the list when it fills (all lanes together), so the
//      warp does not walk the insertion code for every candidate some lane accepts.  The neighbours chosen are exactly
//      those of the definition.  ~300 candidates x 12 instructions per 32 queries instead of ~2,000 instructions per
//      query for a warp per query (measured: profiles/).
//  (b) A free-standing query (far_map_knn_cov: a downsampled scan point against the scan-local map; one query per
//      voxel, nothing to share): one WARP per query, lane l keeps the k smallest of its candidates as a sorted column,
//      then k rounds of warp arg-min over the column heads.
struct __align__(16) Cand {
    double d2;
    uint32_t id;
    uint32_t idx;      // reference bucket * cap + position of the candidate
};

constexpr int LCAP = 24;   // entries of a lane's survivor list

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

// neighbour l of the near-first order: l = 0 the voxel itself, 1..6 face, 7..18 edge, 19..26 corner neighbours;
// packed as (dx + 1) | (dy + 1) << 2 | (dz + 1) << 4
__constant__ uint8_t c_near_first[27] = {
    0x15,
    0x14, 0x16, 0x11, 0x19, 0x05, 0x25,
    0x10, 0x12, 0x18, 0x1A, 0x04, 0x06, 0x24, 0x26, 0x01, 0x09, 0x21, 0x29,
    0x00, 0x02, 0x08, 0x0A, 0x20, 0x22, 0x28, 0x2A};

// R7: mean and centred second moments of the k neighbours in a lane's sorted column, summed in neighbour order, 1/k;
// then Eq. 1.  One lane, FP64.
__device__ __forceinline__ bool column_cov(const MapView& m, const Cand* col, int lane, float cov[6]) {
    const int kk = m.k_cov;
    const double inv_k = 1.0 / (double)kk;
    double mx = 0.0, my = 0.0, mz = 0.0;
    for (int r = 0; r < kk; ++r) {
        const float4 p = __ldg(m.points + col[r * 32 + lane].idx);
        mx += (double)p.x; my += (double)p.y; mz += (double)p.z;
    }
    mx *= inv_k; my *= inv_k; mz *= inv_k;
    double sc[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    for (int r = 0; r < kk; ++r) {
        const float4 p = __ldg(m.points + col[r * 32 + lane].idx);
        const double dx = (double)p.x - mx, dy = (double)p.y - my, dz = (double)p.z - mz;
        sc[0] += dx * dx; sc[1] += dx * dy; sc[2] += dx * dz; sc[3] += dy * dy; sc[4] += dy * dz; sc[5] += dz * dz;
    }
#pragma unroll
    for (int a = 0; a < 6; ++a) sc[a] *= inv_k;
    return regularised_cov(sc, m.cov_eps, cov);
}

// (a) one thread = one query at (qx, qy, qz); `col` = this warp's [k][32] columns, `lst` = its [LCAP][32] survivor lists.
// Returns validity; cov = Eq. 1 or the identity.
// All lanes named in `act` must call together: the walk over the 27 voxels is kept in lockstep (trip counts are the
// warp's maxima) so that the survivor lists are flushed by all lanes at once.
__device__ __noinline__ bool thread_knn_cov_exact(const MapView& m, unsigned act, float qx, float qy, float qz, int lane, Cand* col,
                                                  uint32_t* lst, uint32_t* vox, float cov[6]) {
    const int kk = m.k_cov, cap = m.cap;
    cov[0] = 1.f; cov[1] = 0.f; cov[2] = 0.f; cov[3] = 1.f; cov[4] = 0.f; cov[5] = 1.f;
    int k[3];
    const bool qok = voxel_index(qx, qy, qz, m.voxel, k);      // always true for a stored point
    int cnt = 0, nl = 0;
    float thr = __int_as_float(0x7F800000);            // FP32 bound of the k-th best (+inf until there are k)
    uint32_t* my = lst + lane;
    // exact distance (R6) + sorted insertion of the listed survivors
    auto flush = [&]() {
        for (int e = 0; e < nl; ++e) {
            const uint32_t ref = my[e * 32];
            const float4 p = __ldg(m.points + ref);
            const double d2 = dist2(qx, qy, qz, p.x, p.y, p.z);
            const uint32_t id = __float_as_uint(p.w);
            int q = cnt;
            if (cnt == kk) {
                if (!cand_less(d2, id, col[(kk - 1) * 32 + lane])) continue;
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
            Cand en;
            en.d2 = d2; en.id = id; en.idx = ref;
            col[q * 32 + lane] = en;
        }
        nl = 0;
        if (cnt == kk) thr = __double2float_ru(col[(kk - 1) * 32 + lane].d2) * 1.000001f;
    };
    // pass 1: the 27 table lookups, all in flight at once (they are independent); bucket and count parked in shared memory
    uint32_t* myv = vox + lane;
#pragma unroll 9
    for (int l = 0; l < 27; ++l) {
        const int o = c_near_first[l];
        const int nx = k[0] + (o & 3) - 1, ny = k[1] + ((o >> 2) & 3) - 1, nz = k[2] + ((o >> 4) & 3) - 1;
        uint32_t c = 0, b = 0;
        if (qok && index_in_range(nx) && index_in_range(ny) && index_in_range(nz)) {
            b = find_voxel(m, pack_key(nx, ny, nz), c);
            if (c == 0) b = 0;
        }
        myv[l * 32] = b;
        myv[(27 + l) * 32] = c;
    }
    // pass 2: the candidates, eight loads in flight per lane
    constexpr int U = 8;
    for (int l = 0; l < 27; ++l) {
        const uint32_t b = myv[l * 32], c = myv[(27 + l) * 32];
        const uint32_t cmax = __reduce_max_sync(act, c);
        const float4* bp = m.points + (size_t)b * cap;
        for (uint32_t j0 = 0; j0 < cmax; j0 += U) {
            float4 p[U];
#pragma unroll
            for (int u = 0; u < U; ++u) if (j0 + u < c) p[u] = __ldg(bp + j0 + u);
#pragma unroll
            for (int u = 0; u < U; ++u) {
                if (j0 + u < c) {
                    const float fx = qx - p[u].x, fy = qy - p[u].y, fz = qz - p[u].z;
                    if (fmaf(fz, fz, fmaf(fy, fy, fx * fx)) <= thr) { my[nl * 32] = b * (uint32_t)cap + j0 + u; ++nl; }
                }
            }
            if (__any_sync(act, nl > LCAP - U)) flush();          // all lanes together
        }
    }
    flush();
    if (cnt < kk) return false;                        // fewer than k candidates in the 27 voxels
    float out[6];
    if (!column_cov(m, col, lane, out)) return false;
#pragma unroll
    for (int a = 0; a < 6; ++a) cov[a] = out[a];
    return true;
}

// The fast form of (a) for k <= 10.  A lane keeps its KP = 12 best candidates as ONE 32-bit key each, in registers:
// the FP32 squared distance with its 11 low mantissa bits replaced by the candidate's local index (neighbour 0..26 times
// 64 + position), so unsigned order = distance order (coarsened to 2^-12 relative) and inserting is a branch-free min/max
// chain -- no shared memory, no loop, nothing for the other lanes of the warp to wait for.  The exact FP64 (d2, id)
// selection of R6 then runs on those 12 only.  The result is PROVEN to be the definition's before it is used: a
// candidate that was not kept has a coarse key >= the 12th kept one, hence an exact d2 >= W (1 - 3e-7) with W that key's
// distance bits; if the exact k-th distance is below W (1 - 1e-6) no such candidate can precede it.  Otherwise (a
// near-tie across the 10th..12th neighbour, ~1e-3 of the queries; always on lattice data) the warp redoes its queries
// with thread_knn_cov_exact.
constexpr int KP = 12;
__device__ __forceinline__ bool thread_knn_cov(const MapView& m, unsigned act, float qx, float qy, float qz, int lane, Cand* col,
                                               uint32_t* lst, uint32_t* vox, float cov[6]) {
    const int kk = m.k_cov, cap = m.cap;
    if (kk > KP - 2) return thread_knn_cov_exact(m, act, qx, qy, qz, lane, col, lst, vox, cov);
    cov[0] = 1.f; cov[1] = 0.f; cov[2] = 0.f; cov[3] = 1.f; cov[4] = 0.f; cov[5] = 1.f;
    int k[3];
    const bool qok = voxel_index(qx, qy, qz, m.voxel, k);      // always true for a stored point
    // pass 1: the 27 table lookups, all in flight at once; bucket and count parked in shared memory
    uint32_t* myv = vox + lane;
#pragma unroll 9
    for (int l = 0; l < 27; ++l) {
        const int o = c_near_first[l];
        const int nx = k[0] + (o & 3) - 1, ny = k[1] + ((o >> 2) & 3) - 1, nz = k[2] + ((o >> 4) & 3) - 1;
        uint32_t c = 0, b = 0;
        if (qok && index_in_range(nx) && index_in_range(ny) && index_in_range(nz)) {
            b = find_voxel(m, pack_key(nx, ny, nz), c);
            if (c == 0) b = 0;
        }
        myv[l * 32] = b;
        myv[(27 + l) * 32] = c;
    }
    // pass 2: every candidate -> key -> branch-free insertion into the sorted register array
    uint32_t key[KP];
#pragma unroll
    for (int i = 0; i < KP; ++i) key[i] = 0xFFFFFFFFu;
    constexpr int U = 8;
    for (int l = 0; l < 27; ++l) {
        const uint32_t b = myv[l * 32], c = myv[(27 + l) * 32];
        const float4* bp = m.points + (size_t)b * cap;
        for (uint32_t j0 = 0; j0 < c; j0 += U) {
            float4 p[U];
#pragma unroll
            for (int u = 0; u < U; ++u) if (j0 + u < c) p[u] = __ldg(bp + j0 + u);
#pragma unroll
            for (int u = 0; u < U; ++u) {
                if (j0 + u < c) {
                    const float fx = qx - p[u].x, fy = qy - p[u].y, fz = qz - p[u].z;
                    uint32_t x = (__float_as_uint(fmaf(fz, fz, fmaf(fy, fy, fx * fx))) & 0xFFFFF800u) | ((uint32_t)l << 6) | (j0 + u);
                    if (x < key[KP - 1]) {
#pragma unroll
                        for (int i = 0; i < KP; ++i) { const uint32_t lo = min(key[i], x); x = max(key[i], x); key[i] = lo; }
                    }
                }
            }
        }
    }
    // pass 3: exact (d2, id) order of the kept candidates (R6), through the lane's sorted column in shared memory
    int cnt = 0;
#pragma unroll
    for (int i = 0; i < KP; ++i) {
        if (key[i] != 0xFFFFFFFFu) {
            const uint32_t li = key[i] & 0x7FFu;
            const uint32_t ref = myv[(li >> 6) * 32] * (uint32_t)cap + (li & 63u);
            const float4 p = __ldg(m.points + ref);
            const double d2 = dist2(qx, qy, qz, p.x, p.y, p.z);
            const uint32_t id = __float_as_uint(p.w);
            int q = cnt;
            bool take = true;
            if (cnt == kk) {
                take = cand_less(d2, id, col[(kk - 1) * 32 + lane]);
                q = kk - 1;
            } else {
                ++cnt;
            }
            if (take) {
                while (q > 0) {
                    const Cand c = col[(q - 1) * 32 + lane];
                    if (!cand_less(d2, id, c)) break;
                    col[q * 32 + lane] = c;
                    --q;
                }
                Cand en;
                en.d2 = d2; en.id = id; en.idx = ref;
                col[q * 32 + lane] = en;
            }
        }
    }
    // the proof (see above); fewer than KP candidates in all: nothing was ever rejected
    bool proven = true;
    if (cnt == kk && key[KP - 1] != 0xFFFFFFFFu) {
        const double W = (double)__uint_as_float(key[KP - 1] & 0xFFFFF800u);
        proven = col[(kk - 1) * 32 + lane].d2 < W * (1.0 - 1e-6);
    }
    if (__any_sync(act, !proven)) return thread_knn_cov_exact(m, act, qx, qy, qz, lane, col, lst, vox, cov);
    if (cnt < kk) return false;                        // fewer than k candidates in the 27 voxels
    float out[6];
    if (!column_cov(m, col, lane, out)) return false;
#pragma unroll
    for (int a = 0; a < 6; ++a) cov[a] = out[a];
    return true;
}

__host__ __device__ inline size_t knn_thread_bytes(int k) { return (size_t)32 * k * sizeof(Cand) + (size_t)(LCAP + 54) * 32 * sizeof(uint32_t); }

// queries = stored points named by refs: the points an insert accepted, grouped by voxel
__global__ void __launch_bounds__(256) knn_cov_refs_kernel(MapView m, const uint32_t* __restrict__ refs, const unsigned int* __restrict__ d_n,
                                    int warps_per_block) {
    extern __shared__ __align__(16) char smem[];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    char* wbase = smem + (size_t)wib * knn_thread_bytes(m.k_cov);
    Cand* col = reinterpret_cast<Cand*>(wbase);
    uint32_t* lst = reinterpret_cast<uint32_t*>(wbase + (size_t)32 * m.k_cov * sizeof(Cand));
    uint32_t* vox = lst + LCAP * 32;
    const int64_t n = *d_n;
    const int64_t nwarps = (int64_t)gridDim.x * warps_per_block;
    for (int64_t base = ((int64_t)blockIdx.x * warps_per_block + wib) * 32; base < n; base += nwarps * 32) {
        const int64_t i = base + lane;
        const unsigned act = __ballot_sync(FULL, i < n);
        if (i < n) {
            const uint32_t ref = refs[i];
            const float4 p = m.points[ref];
            float c[6];
            const bool ok = thread_knn_cov(m, act, p.x, p.y, p.z, lane, col, lst, vox, c);
            float* o = m.cov + (size_t)ref * 6;
#pragma unroll
            for (int a = 0; a < 6; ++a) o[a] = c[a];
            m.cov_ok[ref] = ok ? 1 : 0;
        }
    }
}

// same for calls larger than the reference list: every stored point with id >= the call's first id is a new point.
// A warp takes 32 table slots, lists the new points of their voxels in shared memory and serves them 32 at a time.
__global__ void __launch_bounds__(256) knn_cov_new_ids_kernel(MapView m, int warps_per_block) {
    extern __shared__ __align__(16) char smem[];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    char* wbase = smem + (size_t)wib * knn_thread_bytes(m.k_cov);
    Cand* col = reinterpret_cast<Cand*>(wbase);
    uint32_t* lst = reinterpret_cast<uint32_t*>(wbase + (size_t)32 * m.k_cov * sizeof(Cand));
    uint32_t* vox = lst + LCAP * 32;
    const uint32_t first_id = (uint32_t)m.ctr->call_first_id;
    const int64_t nwarps = (int64_t)gridDim.x * warps_per_block;
    for (int64_t s0 = ((int64_t)blockIdx.x * warps_per_block + wib) * 32; s0 < m.slots; s0 += nwarps * 32) {
        Entry e;
        e.key = KEY_EMPTY; e.bucket = NO_BUCKET; e.cr = 0;
        if (s0 + lane < m.slots) e = m.table[s0 + lane];
        uint32_t cnt = entry_count(e.cr), c0 = cnt;
        if (e.key == KEY_EMPTY || e.bucket >= BUCKET_PENDING) cnt = c0 = 0;
        while (c0 > 0 && m.ids[(size_t)e.bucket * m.cap + c0 - 1] >= first_id) --c0;     // ids ascend: the new points are a suffix
        // flatten the warp's new points: lane l's voxel contributes cnt - c0 of them
        const int mine = (int)(cnt - c0);
        const int incl = warp_incl_scan(mine, lane);
        const int total = __shfl_sync(FULL, incl, 31);
        for (int q0 = 0; q0 < total; q0 += 32) {
            const int q = q0 + lane;
            // owner of flattened query q: the lane whose [incl - mine, incl) holds it
            uint32_t ref = 0;
            bool have = false;
            for (int src = 0; src < 32; ++src) {
                const int hi = __shfl_sync(FULL, incl, src), n_src = __shfl_sync(FULL, mine, src);
                const uint32_t b_src = __shfl_sync(FULL, e.bucket, src), c0_src = __shfl_sync(FULL, c0, src);
                if (!have && q < total && q >= hi - n_src && q < hi) { ref = b_src * (uint32_t)m.cap + c0_src + (uint32_t)(q - (hi - n_src)); have = true; }
            }
            const unsigned act = __ballot_sync(FULL, have);
            if (have) {
                const float4 p = m.points[ref];
                float c[6];
                const bool ok = thread_knn_cov(m, act, p.x, p.y, p.z, lane, col, lst, vox, c);
                float* o = m.cov + (size_t)ref * 6;
#pragma unroll
                for (int a = 0; a < 6; ++a) o[a] = c[a];
                m.cov_ok[ref] = ok ? 1 : 0;
            }
            __syncwarp();
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

__host__ __device__ inline size_t knn_warp_bytes(int k) { return (size_t)32 * k * sizeof(Cand) + (size_t)(3 * k + 9) * sizeof(double) + 8 + sizeof(CandList); }

// queries given as points (far_map_knn_cov); n read from the device if d_n != nullptr
__global__ void __launch_bounds__(256, 5) knn_cov_points_kernel(MapView m, const float* __restrict__ q, int64_t n, const int64_t* __restrict__ d_n,
                                      int stride, float* __restrict__ cov6, uint8_t* __restrict__ valid, int warps_per_block) {
    extern __shared__ __align__(16) char smem[];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    char* wbase = smem + (size_t)wib * ((knn_warp_bytes(m.k_cov) + 15) & ~(size_t)15);
    Cand* col = reinterpret_cast<Cand*>(wbase);
    double* mom = reinterpret_cast<double*>(wbase + (size_t)32 * m.k_cov * sizeof(Cand));
    CandList& L = *reinterpret_cast<CandList*>(wbase + (((size_t)32 * m.k_cov * sizeof(Cand) + (size_t)(3 * m.k_cov + 9) * sizeof(double)) + 15 & ~(size_t)15));
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

// The shared-memory opt-in and the occupancy query are slow host calls: done once per (kernel, k_cov, device) and cached
// (the frame chain launches two of these kernels per scan).
template <class K>
static int knn_launch_cfg(const far_map* map, K kernel, size_t per_warp, int64_t work_warps, KnnLaunch& L) {
    struct Cached { bool have; int warps, per_sm; size_t smem; };
    static Cached cache[33][8] = {};          // one table per kernel instantiation
    static size_t attr_bytes[8] = {};         // largest dynamic shared-memory opt-in made for this kernel, per device
    const int dev = map->device & 7;
    Cached& c = cache[map->view.k_cov][dev];
    if (!c.have || map->device >= 8) {
        per_warp = (per_warp + 15) & ~(size_t)15;
        int warps = (int)(100 * 1024 / per_warp);
        if (warps > 8) warps = 8;
        if (warps < 1) warps = 1;
        c.warps = warps;
        c.smem = per_warp * warps;
        c.have = false;
    }
    if (c.smem > attr_bytes[dev]) {           // the opt-in is per function: only ever raise it
        FAR_CUDA(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c.smem));
        attr_bytes[dev] = c.smem;
    }
    if (!c.have) {
        int per_sm = 0;
        FAR_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, c.warps * 32, c.smem));
        c.per_sm = per_sm < 1 ? 1 : per_sm;
        c.have = true;
    }
    L.warps = c.warps; L.smem = c.smem;
    int64_t grid = (int64_t)map->sm_count * c.per_sm;
    const int64_t need = (work_warps + c.warps - 1) / c.warps;
    if (need < grid) grid = need;
    if (grid < 1) grid = 1;
    L.grid = (int)grid;
    return FAR_OK;
}

int launch_knn_cov_refs(const far_map* map, const uint32_t* d_refs, const unsigned int* d_n, int64_t n_max, cudaStream_t st) {
    KnnLaunch L;
    int rc = knn_launch_cfg(map, knn_cov_refs_kernel, knn_thread_bytes(map->view.k_cov), (n_max + 31) / 32, L);
    if (rc != FAR_OK) return rc;
    FAR_LAUNCH(knn_cov_refs_kernel, L.grid, L.warps * 32, L.smem, st, map->view, d_refs, d_n, L.warps);
    FAR_CUDA(cudaGetLastError());
    return FAR_OK;
}

int launch_knn_cov_new_ids(const far_map* map, cudaStream_t st) {
    KnnLaunch L;
    int rc = knn_launch_cfg(map, knn_cov_new_ids_kernel, knn_thread_bytes(map->view.k_cov), (map->view.slots + 31) / 32, L);
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
        int v = 0;
        FAR_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&v, nn_kernel, QWARPS * 32, 0));
        per_sm = v < 1 ? 1 : v;
    }
    int64_t grid = (int64_t)map->sm_count * per_sm;
    const int64_t need = (m + QWARPS - 1) / QWARPS;
    if (need < grid) grid = need;
    FAR_LAUNCH(nn_kernel, (int)grid, QWARPS * 32, 0, (cudaStream_t)stream, map->view, d_q, m, stride, d_id, d_d2);
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
    int rc = knn_launch_cfg(map, knn_cov_points_kernel, knn_warp_bytes(map->view.k_cov), m, L);
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
