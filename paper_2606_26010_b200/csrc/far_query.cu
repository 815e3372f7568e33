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
                                                               int32_t* __restrict__ out) {
    __shared__ CandList s_list[QWARPS];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const int64_t nwarps = (int64_t)gridDim.x * QWARPS;
    for (int64_t i = (int64_t)blockIdx.x * QWARPS + wib; i < n; i += nwarps) {
        const float* qq = q + i * stride;
        int k[3];
        int total = 0;
        if (voxel_index(__ldg(qq), __ldg(qq + 1), __ldg(qq + 2), m.voxel, k)) total = probe27(m, k, lane, s_list[wib]);
        if (lane == 0) out[i] = total;
        __syncwarp();
    }
}

// ---- A7: k nearest by (d2, id) -> Eq. 1 -----------------------------------------------------------------------
// Selection without a sort of all candidates: every lane keeps the k smallest of ITS candidates as a sorted
// column in shared memory (insertion while the candidates stream in; a candidate that cannot enter the lane's
// top k costs one comparison).  The k nearest overall are then k rounds of a warp arg-min over the column heads;
// the winning lane just advances its head.  Shared memory per warp: 32 lanes x k x 16 B, independent of cap.
struct __align__(16) Cand {
    double d2;
    uint32_t id;
    uint32_t ref;
};

__host__ __device__ inline size_t knn_smem_per_warp(int k) { return (size_t)32 * k * sizeof(Cand) + sizeof(CandList); }

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

// one query by one warp; all lanes return the same (valid, cov)
__device__ __forceinline__ bool warp_knn_cov(const MapView& m, float qx, float qy, float qz, int lane, char* smem_w,
                                             float cov[6]) {
    const int cap = m.cap, kk = m.k_cov;
    Cand* col = reinterpret_cast<Cand*>(smem_w);                 // col[r * 32 + lane] = r-th smallest of this lane
    CandList& L = *reinterpret_cast<CandList*>(smem_w + (size_t)32 * kk * sizeof(Cand));
    cov[0] = 1.f; cov[1] = 0.f; cov[2] = 0.f; cov[3] = 1.f; cov[4] = 0.f; cov[5] = 1.f;
    int k[3];
    if (!voxel_index(qx, qy, qz, m.voxel, k)) return false;
    const int total = probe27(m, k, lane, L);
    if (total < kk) { __syncwarp(); return false; }
    const double INF = __longlong_as_double(0x7FF0000000000000ll);
    const double dqx = (double)qx, dqy = (double)qy, dqz = (double)qz;
    int cnt = 0;
    CandIter ci;
    ci.before = 0;
    for (int j = lane, step = 0; j < total; j += 32, ++step) {
        const uint32_t ref = cand_next(L, ci, step, j, lane, cap);
        const float4 p = __ldg(m.points + ref);
        const double dx = dqx - (double)p.x, dy = dqy - (double)p.y, dz = dqz - (double)p.z;
        const double d2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));   // R6
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
        e.d2 = d2; e.id = id; e.ref = ref;
        col[q * 32 + lane] = e;
    }
    // k rounds of warp arg-min over the column heads
    int h = 0;
    Cand head;
    head.d2 = INF; head.id = NO_ID; head.ref = 0;
    if (cnt > 0) head = col[lane];
    uint32_t myref = 0;
    for (int r = 0; r < kk; ++r) {
        const int w = warp_argmin(head.d2, head.id);
        const uint32_t wref = __shfl_sync(FULL, head.ref, w);
        if (lane == r) myref = wref;
        if (lane == w) {
            ++h;
            if (h < cnt) head = col[h * 32 + lane];
            else { head.d2 = INF; head.id = NO_ID; }
        }
    }
    // lane r < k holds the r-th neighbour.  The neighbours go through shared memory (the candidate columns are no
    // longer needed) so that the moments are computed once, not by 32 lanes in lockstep through shuffles: lane a < 3
    // sums coordinate a in neighbour order (R7: 1/k), then lane a < 6 accumulates centred product a, also in order.
    __syncwarp();
    double* nb = reinterpret_cast<double*>(smem_w);          // [kk][3] positions, then [3] mean, then [6] moments
    if (lane < kk) {
        const float4 p = __ldg(m.points + myref);
        nb[3 * lane] = (double)p.x; nb[3 * lane + 1] = (double)p.y; nb[3 * lane + 2] = (double)p.z;
    }
    __syncwarp();
    const double inv_k = 1.0 / (double)kk;
    double* mean = nb + 3 * kk;
    double* mom = mean + 3;
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
        mom[lane] = sacc * inv_k;
    }
    __syncwarp();
    double sc[6];
#pragma unroll
    for (int a = 0; a < 6; ++a) sc[a] = mom[a];
    __syncwarp();
    float out[6];
    if (!regularised_cov(sc, m.cov_eps, out)) return false;
#pragma unroll
    for (int a = 0; a < 6; ++a) cov[a] = out[a];
    return true;
}

// queries given as points (far_map_knn_cov); n read from the device if d_n != nullptr
__global__ void __launch_bounds__(256, 5) knn_cov_points_kernel(MapView m, const float* __restrict__ q, int64_t n, const int64_t* __restrict__ d_n,
                                      int stride, float* __restrict__ cov6, uint8_t* __restrict__ valid, int warps_per_block) {
    extern __shared__ __align__(16) char smem[];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    char* smem_w = smem + (size_t)wib * knn_smem_per_warp(m.k_cov);
    if (d_n) n = min(n, *d_n);
    const int64_t nwarps = (int64_t)gridDim.x * warps_per_block;
    for (int64_t i = (int64_t)blockIdx.x * warps_per_block + wib; i < n; i += nwarps) {
        const float* qq = q + i * stride;
        float c[6];
        const bool ok = warp_knn_cov(m, __ldg(qq), __ldg(qq + 1), __ldg(qq + 2), lane, smem_w, c);
        if (lane < 6) cov6[i * 6 + lane] = c[lane];
        if (lane == 0) valid[i] = ok ? 1 : 0;
    }
}

// queries = the points an insert accepted, one task per touched voxel: bucket, first new position, count
__global__ void __launch_bounds__(256, 5) knn_cov_tasks_kernel(MapView m, const uint2* __restrict__ tasks, const unsigned int* __restrict__ d_n,
                                    int warps_per_block) {
    extern __shared__ __align__(16) char smem[];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    char* smem_w = smem + (size_t)wib * knn_smem_per_warp(m.k_cov);
    const int64_t n = *d_n;
    const int64_t nwarps = (int64_t)gridDim.x * warps_per_block;
    for (int64_t i = (int64_t)blockIdx.x * warps_per_block + wib; i < n; i += nwarps) {
        const uint2 t = tasks[i];
        const uint32_t c0 = t.y & 0xFFu, n_new = t.y >> 8;
        for (uint32_t j = c0; j < c0 + n_new; ++j) {
            const uint32_t ref = t.x * (uint32_t)m.cap + j;
            const float4 p = m.points[ref];
            float c[6];
            const bool ok = warp_knn_cov(m, p.x, p.y, p.z, lane, smem_w, c);
            if (lane < 6) m.cov[(size_t)ref * 6 + lane] = c[lane];
            if (lane == 0) m.cov_ok[ref] = ok ? 1 : 0;
        }
    }
}

// same for calls larger than the task list: every stored point with id >= the call's first id is a new point
__global__ void __launch_bounds__(256, 5) knn_cov_new_ids_kernel(MapView m, int warps_per_block) {
    extern __shared__ __align__(16) char smem[];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    char* smem_w = smem + (size_t)wib * knn_smem_per_warp(m.k_cov);
    const uint32_t first_id = (uint32_t)m.ctr->call_first_id;
    const int64_t nwarps = (int64_t)gridDim.x * warps_per_block;
    for (int64_t s = (int64_t)blockIdx.x * warps_per_block + wib; s < m.slots; s += nwarps) {
        const Entry e = m.table[s];
        const uint32_t cnt = entry_count(e.cr);
        if (e.key == KEY_EMPTY || e.bucket >= BUCKET_PENDING || cnt == 0) continue;
        for (uint32_t j = 0; j < cnt; ++j) {
            const uint32_t ref = e.bucket * (uint32_t)m.cap + j;
            const float4 p = m.points[ref];
            if (__float_as_uint(p.w) < first_id) continue;
            float c[6];
            const bool ok = warp_knn_cov(m, p.x, p.y, p.z, lane, smem_w, c);
            if (lane < 6) m.cov[(size_t)ref * 6 + lane] = c[lane];
            if (lane == 0) m.cov_ok[ref] = ok ? 1 : 0;
        }
    }
}

struct KnnLaunch { int warps, grid; size_t smem; };

// The shared-memory opt-in and the occupancy query are slow host calls: done once per (kernel, k_cov, device) and cached
// (the frame chain launches two of these kernels per scan and is host-enqueue-bound end to end).
template <class K>
static int knn_launch_cfg(const far_map* map, K kernel, int64_t work, KnnLaunch& L) {
    struct Cached { bool have; int warps, per_sm; size_t smem; };
    static Cached cache[33][8] = {};          // one table per kernel instantiation
    const int dev = map->device & 7;
    Cached& c = cache[map->view.k_cov][dev];
    static size_t attr_bytes[8] = {};         // largest dynamic shared-memory opt-in made for this kernel, per device
    if (c.have && map->device < 8) {
        L.warps = c.warps; L.smem = c.smem;
        if (c.smem > attr_bytes[dev]) {       // another k_cov lowered nothing, but a larger one may be needed now
            FAR_CUDA(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c.smem));
            attr_bytes[dev] = c.smem;
        }
        int64_t grid = (int64_t)map->sm_count * c.per_sm;
        const int64_t need = (work + c.warps - 1) / c.warps;
        if (need < grid) grid = need;
        if (grid < 1) grid = 1;
        L.grid = (int)grid;
        return FAR_OK;
    }
    const size_t per_warp = knn_smem_per_warp(map->view.k_cov);
    int warps = (int)(100 * 1024 / per_warp);
    if (warps > 8) warps = 8;
    if (warps < 1) warps = 1;
    L.warps = warps;
    L.smem = per_warp * warps;
    if (L.smem > attr_bytes[dev]) {           // the opt-in is per function: only ever raise it
        FAR_CUDA(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L.smem));
        attr_bytes[dev] = L.smem;
    }
    int per_sm = 0;
    FAR_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, warps * 32, L.smem));
    if (per_sm < 1) per_sm = 1;
    c.warps = warps; c.per_sm = per_sm; c.smem = L.smem; c.have = true;
    int64_t grid = (int64_t)map->sm_count * per_sm;
    const int64_t need = (work + warps - 1) / warps;
    if (need < grid) grid = need;
    if (grid < 1) grid = 1;
    L.grid = (int)grid;
    return FAR_OK;
}

int launch_knn_cov_tasks(const far_map* map, const uint2* d_tasks, const unsigned int* d_n, int64_t n_max, cudaStream_t st) {
    KnnLaunch L;
    int rc = knn_launch_cfg(map, knn_cov_tasks_kernel, n_max, L);
    if (rc != FAR_OK) return rc;
    FAR_LAUNCH(knn_cov_tasks_kernel, L.grid, L.warps * 32, L.smem, st, map->view, d_tasks, d_n, L.warps);
    FAR_CUDA(cudaGetLastError());
    return FAR_OK;
}

int launch_knn_cov_new_ids(const far_map* map, cudaStream_t st) {
    KnnLaunch L;
    int rc = knn_launch_cfg(map, knn_cov_new_ids_kernel, map->view.slots, L);
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

int far_map_count27(const far_map_t* map, const float* d_q, int64_t m, int stride, int32_t* d_count, void* stream) {
    if (!map || m < 0 || (stride != 3 && stride != 4) || (m > 0 && (!d_q || !d_count))) return FAR_ERR_ARG;
    if (m == 0) return FAR_OK;
    int64_t grid = (int64_t)map->sm_count * 8;
    const int64_t need = (m + QWARPS - 1) / QWARPS;
    if (need < grid) grid = need;
    FAR_LAUNCH(count27_kernel, (int)grid, QWARPS * 32, 0, (cudaStream_t)stream, map->view, d_q, m, stride, d_count);
    FAR_CUDA(cudaGetLastError());
    return FAR_OK;
}

static int knn_cov_impl(const far_map_t* map, const float* d_q, int64_t m, const int64_t* d_m, int stride, float* d_cov6,
                        uint8_t* d_valid, void* stream) {
    if (!map || m < 0 || (stride != 3 && stride != 4) || (m > 0 && (!d_q || !d_cov6 || !d_valid))) return FAR_ERR_ARG;
    if (m == 0) return FAR_OK;
    KnnLaunch L;
    int rc = knn_launch_cfg(map, knn_cov_points_kernel, m, L);
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
