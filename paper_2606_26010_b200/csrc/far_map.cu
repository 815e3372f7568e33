// far_map.cu -- the voxel hashmap: create / clear / deterministic capped insert / prune / export / stats.
//
// PAPER.md:62-68 (cuVoxelMap: custom key = 3D voxel indices, linear probing, <= N_max points per voxel, built
// for concurrent access), PAPER.md:109 (submap update: insert at T_L with a per-voxel cap, recompute the
// covariances of added points only, remove voxels beyond a range limit).
//
// Deterministic capped insert (reading R3: the result equals inserting the points one by one in index order).
// A bare atomicAdd ticket gives the right counts but timing-dependent contents, so instead each offered point
// runs an *atomicMin insertion chain* on the id words of its voxel's free positions c0..cap-1 (all FAR_NO_ID =
// +inf before the batch):   x = my id;  for pos = c0..cap-1:  old = atomicMin(&id[pos], x);
//                           old == NO_ID -> placed, stop;   old > x -> carry the displaced id: x = old.
// Every id of the batch that targets the voxel enters at position c0 and every id except the final occupant of
// a position moves on to the next one exactly once, so position c0+r ends up holding the (r+1)-th smallest id
// whatever the interleaving: the lowest ids win, in ascending order, with no sort.  Ids already stored are all
// smaller than the batch's ids (ids grow monotonically), so they stay where they are.  A second kernel walks
// the voxels that received a point, fetches the coordinates of the surviving ids (index = id - first id of
// the chunk) and writes them next to their id.
#include <cstdio>
#include <cstring>
#include <new>

#include "far_internal.h"

using namespace far;

namespace far {

static thread_local char g_cuda_err[256] = "";
void set_cuda_error(cudaError_t e, const char* where) {
    snprintf(g_cuda_err, sizeof(g_cuda_err), "%s: %s (%s)", cudaGetErrorName(e), cudaGetErrorString(e), where);
}

__device__ __forceinline__ bool load_pose_point(const float* __restrict__ xyz, int64_t i, int stride, int pose_mode,
                                                const Pose& T, float p[3]) {
    const float* s = xyz + i * stride;
    const float x = s[0], y = s[1], z = s[2];
    if (!(isfinite(x) && isfinite(y) && isfinite(z))) return false;
    if (pose_mode) transform_point(T, x, y, z, p);
    else { p[0] = x; p[1] = y; p[2] = z; }
    return true;
}

// ---- Adaptive Submap Density (R17) -----------------------------------------------------
// per-voxel limit N_ASMD = clamp(floor(n_close (1 - d/d_max) + 0.5), k_cov, cap), d = distance of the voxel centre
// from the current pose; every operation one rounded binary64 operation so that the integer it decides is the
// oracle's.  `on == 0`: the fixed cap (plain far_map_insert).
struct Asmd {
    const double* d_n_close;   // device: mean points per voxel near the scan (far_asmd_density)
    double d_max;
    int on;
};

__device__ __forceinline__ uint32_t voxel_limit(const MapView& m, const Asmd& A, const int k[3], int pose_mode, const Pose& T) {
    if (!A.on) return (uint32_t)m.cap;
    const double v = (double)m.voxel;
    const double cx = pose_mode ? T.t[0] : 0.0, cy = pose_mode ? T.t[1] : 0.0, cz = pose_mode ? T.t[2] : 0.0;
    const double dx = __dadd_rn(__dmul_rn(__dadd_rn((double)k[0], 0.5), v), -cx);
    const double dy = __dadd_rn(__dmul_rn(__dadd_rn((double)k[1], 0.5), v), -cy);
    const double dz = __dadd_rn(__dmul_rn(__dadd_rn((double)k[2], 0.5), v), -cz);
    const double d = __dsqrt_rn(__dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz)));
    const double f = __dadd_rn(1.0, -__ddiv_rn(d, A.d_max));
    const double x = floor(__dadd_rn(__dmul_rn(__ldg(A.d_n_close), f), 0.5));
    const double lo = (double)m.k_cov, hi = (double)m.cap;
    uint32_t lim = (uint32_t)m.k_cov;
    if (x > lo) lim = (x >= hi) ? (uint32_t)m.cap : (uint32_t)x;
    return min(lim, (uint32_t)m.cap);
}

// ---- insert, kernel 1: key -> find-or-claim -> atomicMin chain ---------------------------------------
__global__ void __launch_bounds__(256) insert_claim_chain_kernel(MapView m, const float* __restrict__ xyz, int64_t n,
                                                                  int stride, int pose_mode, Pose hpose,
                                                                  const Pose* __restrict__ d_pose, uint32_t first_id,
                                                                  uint32_t* __restrict__ touched, Asmd asmd) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const Pose& T = (pose_mode == 2) ? *d_pose : hpose;
    // the key count is read once, up front (its latency hides behind the point load); the limit is enforced up to the
    // keys claimed while this kernel runs -- which excess voxels are dropped is unspecified anyway (R3)
    const unsigned long long keys_before = *reinterpret_cast<volatile unsigned long long*>(&m.ctr->n_keys);
    float p[3];
    int k[3];
    if (!load_pose_point(xyz, i, stride, pose_mode, T, p) || !voxel_index(p[0], p[1], p[2], m.voxel, k)) {
        atomicAdd(&m.ctr->st_invalid, 1ull);
        return;
    }
    const unsigned long long key = pack_key(k[0], k[1], k[2]);
    // Lanes of this warp that offer points to the SAME voxel (a LiDAR ring crossing a voxel gives a run of consecutive
    // ids; 73 % of a C2 scan falls into voxels that are offered more than cap points, up to 700).  Ids grow with the
    // lane, so `ahead` of them are smaller than mine: my final position is at least c0 + ahead.  Entering the chain
    // there instead of at c0 is exact (an id may enter anywhere at or before its final position: every position still
    // ends up with the minimum of the ids that reach it) and removes most of the shifting; if c0 + ahead is already
    // past the limit the point cannot survive at all.
    const unsigned same = __match_any_sync(__activemask(), key);
    const uint32_t ahead = __popc(same & ((1u << (threadIdx.x & 31)) - 1u));
    // find or claim the voxel's slot: 64-bit atomicCAS on the key word, linear probing step 1
    uint32_t s = hash_key(key) & m.mask;
    bool found = false, new_key = false;
    for (uint32_t probes = 0; probes < m.slots; ++probes) {
        unsigned long long cur = *reinterpret_cast<volatile unsigned long long*>(&m.table[s].key);
        if (cur == KEY_EMPTY) {
            if (keys_before >= m.max_keys) break;   // table full
            cur = atomicCAS(&m.table[s].key, KEY_EMPTY, key);
            if (cur == KEY_EMPTY) {
                new_key = true;
                found = true;
                // keep the reach of the key's home slot up to date (far_common.cuh::find_voxel)
                atomicMax(&m.table[hash_key(key) & m.mask].pad, probes + 1u);
                break;
            }
        }
        if (cur == key) { found = true; break; }
        s = (s + 1) & m.mask;
    }
    if (new_key) {
        // one atomic per group of lanes that claimed a key together, not one per key: tens of thousands of
        // same-address atomics per scan serialise in a single L2 slice (C4: 72k per 100k-point batch)
        const unsigned grp = __activemask();
        if ((threadIdx.x & 31) == __ffs(grp) - 1) atomicAdd(&m.ctr->n_keys, (unsigned long long)__popc(grp));
    }
    if (!found) {
        atomicAdd(&m.ctr->st_dropped_full, 1ull);
        m.ctr->full_flag = 1u;
        return;
    }
    // count is only written by the commit kernel, so it is stable here: c0 = points stored before this chunk
    const uint32_t c0 = *reinterpret_cast<volatile uint32_t*>(&m.table[s].count);
    // cap = this voxel's limit: the fixed cap, or N_ASMD (positions at and beyond it are never written)
    const uint32_t cap = voxel_limit(m, asmd, k, pose_mode, T);
    if (c0 + ahead >= cap) return;
    uint32_t* idw = m.ids + (size_t)s * (uint32_t)m.cap;   // id word of position 0 (compact array)
    uint32_t x = first_id + (uint32_t)i;
    // ids at a position only ever decrease: if the last position already holds a smaller id, x cannot survive
    const uint32_t last = *reinterpret_cast<volatile uint32_t*>(idw + (cap - 1));
    if (last < x) return;
    // The id words of a bucket are sorted at every instant and only ever decrease, so a position seen holding an
    // id < x will never take x: gallop over such positions with plain reads (4 independent loads per step)
    // instead of walking them with dependent atomics.  A stale read only makes the chain start earlier.
    uint32_t pos = c0 + ahead;
    while (pos + 4 <= cap) {
        const uint32_t a3 = *reinterpret_cast<volatile uint32_t*>(idw + (pos + 3));
        if (a3 < x) pos += 4; else break;
    }
    for (; pos < cap; ++pos) {
        const uint32_t old = atomicMin(idw + pos, x);
        if (old == NO_ID) {
            if (pos == c0) touched[atomicAdd(&m.ctr->n_touched, 1u)] = s;   // unique per voxel and chunk
            break;
        }
        if (old > x) x = old;
    }
}

// ---- insert, kernel 2: 8 lanes per touched voxel write the coordinates of the surviving ids -------------------
// Every step of a voxel's commit is a dependent, usually cold access (touched list -> entry -> id row -> source point ->
// bucket), and most touched voxels receive a handful of points, so a warp works on FOUR voxels at once: four times the
// memory-level parallelism of a warp per voxel (C4, where almost every point opens its own voxel in a multi-GB pool,
// is bound by exactly that).  The statistics are accumulated per warp and flushed once at the end.
constexpr int COMMIT_LANES = 8;      // 4 and 16 measure the same within 3 %
__global__ void __launch_bounds__(256) insert_commit_kernel(MapView m, const float* __restrict__ xyz, int stride,
                                                             int pose_mode, Pose hpose, const Pose* __restrict__ d_pose,
                                                             uint32_t first_id, const uint32_t* __restrict__ touched,
                                                             uint32_t* __restrict__ cov_list, int64_t cov_list_cap) {
    const int lane = threadIdx.x & 31, sub = lane / COMMIT_LANES, sl = lane % COMMIT_LANES;
    constexpr int PER_WARP = 32 / COMMIT_LANES;
    const unsigned gmask = ((1u << COMMIT_LANES) - 1u) << (sub * COMMIT_LANES);
    const int64_t warp = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int64_t nwarps = ((int64_t)gridDim.x * blockDim.x) >> 5;
    const Pose& T = (pose_mode == 2) ? *d_pose : hpose;
    const uint32_t n_touched = m.ctr->n_touched;
    const uint32_t cap = (uint32_t)m.cap;
    unsigned long long acc_new = 0, acc_vox = 0;          // lane sl == 0 of each group: points accepted, voxels opened
    for (int64_t t0 = warp * PER_WARP; t0 < n_touched; t0 += nwarps * PER_WARP) {
        const int64_t t = t0 + sub;
        const bool active = t < n_touched;
        uint32_t s = 0, c0 = cap;
        if (active) {
            s = touched[t];
            c0 = m.table[s].count;
        }
        uint32_t n_new = 0;
        for (uint32_t step = 0; step * COMMIT_LANES < cap; ++step) {      // warp-uniform trip count
            const uint32_t pos = c0 + step * COMMIT_LANES + sl;
            uint32_t id = NO_ID;
            if (active && pos < cap) id = m.ids[(size_t)s * cap + pos];
            const bool is_new = id != NO_ID;
            if (is_new) {
                float p[3];
                load_pose_point(xyz, (int64_t)(id - first_id), stride, pose_mode, T, p);
                m.points[(size_t)s * cap + pos] = make_float4(p[0], p[1], p[2], __uint_as_float(id));
                if (m.cov_ok) m.cov_ok[(size_t)s * cap + pos] = 0;
            }
            const unsigned b = __ballot_sync(FULL, is_new);
            if (b == 0) break;                                             // ids fill positions in order: nothing further
            if (cov_list != nullptr) {
                uint32_t at = 0;
                if (lane == 0) at = atomicAdd(&m.ctr->n_cov, (uint32_t)__popc(b));
                at = __shfl_sync(FULL, at, 0);
                const uint32_t mine = at + __popc(b & ((1u << lane) - 1u));
                if (is_new && mine < cov_list_cap) cov_list[mine] = s * cap + pos;
            }
            n_new += __popc(b & gmask);
        }
        if (active && sl == 0) {
            m.table[s].count = c0 + n_new;
            acc_new += n_new;
            if (c0 == 0) acc_vox += 1;
        }
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        acc_new += __shfl_xor_sync(FULL, acc_new, d);
        acc_vox += __shfl_xor_sync(FULL, acc_vox, d);
    }
    if (lane == 0) {
        if (acc_new) atomicAdd(&m.ctr->st_accepted, acc_new);
        if (acc_vox) atomicAdd(&m.ctr->st_new_voxels, acc_vox);
    }
}

__global__ void insert_stats_kernel(MapView m, int64_t n_offered, far_insert_stats_t* out) {
    if (threadIdx.x == 0 && blockIdx.x == 0 && out) {
        out->n_offered = n_offered;
        out->n_accepted = (int64_t)m.ctr->st_accepted;
        out->n_new_voxels = (int64_t)m.ctr->st_new_voxels;
        out->n_dropped_full = (int64_t)m.ctr->st_dropped_full;
        out->n_invalid = (int64_t)m.ctr->st_invalid;
    }
}

// ---- A5 prune (R5): thread per slot, FP64 squared centre distance, strict > -------------------
__global__ void __launch_bounds__(256) prune_kernel(MapView m, double cx, double cy, double cz, const Pose* d_pose,
                                                     double r2, far_prune_stats_t* __restrict__ out) {
    const uint32_t s = blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long vr = 0, pr = 0, vl = 0, pl = 0;
    if (s < m.slots) {
        const Entry e = m.table[s];
        if (e.key != KEY_EMPTY && e.count > 0) {
            if (d_pose) { cx = d_pose->t[0]; cy = d_pose->t[1]; cz = d_pose->t[2]; }
            int k[3];
            unpack_key(e.key, k);
            const double v = (double)m.voxel;
            const double dx = __dadd_rn(__dmul_rn(__dadd_rn((double)k[0], 0.5), v), -cx);
            const double dy = __dadd_rn(__dmul_rn(__dadd_rn((double)k[1], 0.5), v), -cy);
            const double dz = __dadd_rn(__dmul_rn(__dadd_rn((double)k[2], 0.5), v), -cz);
            const double d2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
            if (d2 > r2) {
                // the key stays (dead key, count 0); its id words go back to +inf so a later insert starts clean
                for (uint32_t j = 0; j < e.count; ++j) {
                    m.ids[(size_t)s * m.cap + j] = NO_ID;
                    if (m.cov_ok) m.cov_ok[(size_t)s * m.cap + j] = 0;
                }
                m.table[s].count = 0;
                vr = 1; pr = e.count;
            } else {
                vl = 1; pl = e.count;
            }
        }
    }
    // block-aggregate the four statistics: one atomic per counter and block (the four words are a hot spot)
    __shared__ unsigned long long s_acc[8][4];
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        vr += __shfl_xor_sync(FULL, vr, d); pr += __shfl_xor_sync(FULL, pr, d);
        vl += __shfl_xor_sync(FULL, vl, d); pl += __shfl_xor_sync(FULL, pl, d);
    }
    if ((threadIdx.x & 31) == 0) {
        s_acc[threadIdx.x >> 5][0] = vr; s_acc[threadIdx.x >> 5][1] = pr;
        s_acc[threadIdx.x >> 5][2] = vl; s_acc[threadIdx.x >> 5][3] = pl;
    }
    __syncthreads();
    if (threadIdx.x < 4) {
        unsigned long long t = 0;
#pragma unroll
        for (int w = 0; w < 8; ++w) t += s_acc[w][threadIdx.x];
        if (t) atomicAdd(&m.ctr->pr_vox_removed + threadIdx.x, t);
        __threadfence();
    }
    // the block that takes the last ticket writes the statistics out and re-arms the counters: no second launch
    __shared__ bool s_last;
    __syncthreads();
    if (threadIdx.x == 0) s_last = atomicAdd(&m.ctr->pad, 1u) == gridDim.x - 1;
    __syncthreads();
    if (s_last && threadIdx.x == 0) {
        __threadfence();
        volatile unsigned long long* c = &m.ctr->pr_vox_removed;
        if (out) {
            out->n_voxels_removed = (int64_t)c[0];
            out->n_points_removed = (int64_t)c[1];
            out->n_voxels_left = (int64_t)c[2];
            out->n_points_left = (int64_t)c[3];
        }
        c[0] = 0ull; c[1] = 0ull; c[2] = 0ull; c[3] = 0ull;
        m.ctr->pad = 0u;
    }
}

// ---- ASMD density (R17): integer sums over the live voxels near the centre, one division at the end --
__global__ void __launch_bounds__(256) asmd_density_kernel(MapView m, double cx, double cy, double cz, double r2,
                                                            unsigned long long* acc /* [2]: voxels, points */) {
    const uint32_t s = blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long nv = 0, np = 0;
    if (s < m.slots) {
        const Entry e = m.table[s];
        if (e.key != KEY_EMPTY && e.count > 0) {
            int k[3];
            unpack_key(e.key, k);
            const double v = (double)m.voxel;
            const double dx = __dadd_rn(__dmul_rn(__dadd_rn((double)k[0], 0.5), v), -cx);
            const double dy = __dadd_rn(__dmul_rn(__dadd_rn((double)k[1], 0.5), v), -cy);
            const double dz = __dadd_rn(__dmul_rn(__dadd_rn((double)k[2], 0.5), v), -cz);
            const double d2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
            if (d2 <= r2) { nv = 1; np = e.count; }
        }
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) { nv += __shfl_xor_sync(FULL, nv, d); np += __shfl_xor_sync(FULL, np, d); }
    if ((threadIdx.x & 31) == 0 && nv) { atomicAdd(&acc[0], nv); atomicAdd(&acc[1], np); }
}

__global__ void asmd_density_out_kernel(MapView m, const unsigned long long* acc, double* out) {
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        out[0] = acc[0] ? __ddiv_rn((double)acc[1], (double)acc[0]) : (double)m.cap;
        out[1] = (double)acc[0];
    }
}

// ---- clear: reset only what is in use (the pool itself is never touched beyond the live buckets) ------------
__global__ void __launch_bounds__(256) clear_kernel(MapView m) {
    const uint32_t s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= m.slots) return;
    const Entry e = m.table[s];
    if (e.key == KEY_EMPTY) return;
    for (uint32_t j = 0; j < e.count; ++j) m.ids[(size_t)s * m.cap + j] = NO_ID;
    Entry z;
    z.key = KEY_EMPTY; z.count = 0; z.pad = 0;
    m.table[s] = z;
}

__global__ void __launch_bounds__(256) table_init_kernel(Entry* table, uint32_t slots) {
    const uint32_t s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= slots) return;
    Entry z;
    z.key = KEY_EMPTY; z.count = 0; z.pad = 0;
    table[s] = z;
}

// ---- stats / export ----------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) stats_kernel(MapView m, unsigned long long* acc /* [3] */) {
    const uint32_t s = blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long nv = 0, np = 0, nd = 0;
    if (s < m.slots) {
        const Entry e = m.table[s];
        if (e.key != KEY_EMPTY) {
            if (e.count > 0) { nv = 1; np = e.count; } else nd = 1;
        }
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        nv += __shfl_xor_sync(FULL, nv, d); np += __shfl_xor_sync(FULL, np, d); nd += __shfl_xor_sync(FULL, nd, d);
    }
    if ((threadIdx.x & 31) == 0 && (nv | nd)) {
        if (nv) { atomicAdd(&acc[0], nv); atomicAdd(&acc[1], np); }
        if (nd) atomicAdd(&acc[2], nd);
    }
}

__global__ void stats_out_kernel(MapView m, unsigned long long* acc, unsigned long long next_id, far_map_stats_t* out) {
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        out->n_voxels = (int64_t)acc[0];
        out->n_points = (int64_t)acc[1];
        out->n_dead_keys = (int64_t)acc[2];
        out->n_slots = (int64_t)m.slots;
        out->next_id = next_id;
        acc[0] = acc[1] = acc[2] = 0ull;
    }
}

// one warp per group of 32 slots; live voxels get consecutive output rows (order unspecified)
__global__ void __launch_bounds__(256) export_kernel(MapView m, unsigned long long* __restrict__ keys,
                                                      int32_t* __restrict__ counts, float4* __restrict__ pts,
                                                      float* __restrict__ cov6, uint8_t* __restrict__ cov_ok,
                                                      int64_t max_out, unsigned long long* n_out) {
    const int lane = threadIdx.x & 31;
    const uint32_t s = blockIdx.x * blockDim.x + threadIdx.x;
    Entry e;
    e.key = KEY_EMPTY; e.count = 0;
    if (s < m.slots) e = m.table[s];
    const bool live = e.key != KEY_EMPTY && e.count > 0;
    const unsigned b = __ballot_sync(FULL, live);
    if (!b) return;
    unsigned long long base = 0;
    if (lane == 0) base = atomicAdd(n_out, (unsigned long long)__popc(b));
    base = __shfl_sync(FULL, base, 0);
    const unsigned long long row = base + __popc(b & ((1u << lane) - 1u));
    if (live && (int64_t)row < max_out) {
        keys[row] = e.key;
        counts[row] = (int32_t)e.count;
    }
    // cooperative copy of each live bucket of this warp
    unsigned rem = b;
    while (rem) {
        const int src = __ffs(rem) - 1;
        rem &= rem - 1;
        const uint32_t ss = (blockIdx.x * blockDim.x + (threadIdx.x & ~31)) + src;
        const uint32_t cnt = __shfl_sync(FULL, e.count, src);
        const unsigned long long r = __shfl_sync(FULL, row, src);
        if ((int64_t)r >= max_out) continue;
        for (uint32_t j = lane; j < (uint32_t)m.cap; j += 32) {
            const bool have = j < cnt;
            const size_t from = (size_t)ss * m.cap + j, to = (size_t)r * m.cap + j;
            if (pts) pts[to] = have ? m.points[from] : make_float4(0.f, 0.f, 0.f, __uint_as_float(NO_ID));
            if (cov6) {
                for (int a = 0; a < 6; ++a) cov6[to * 6 + a] = (have && m.cov) ? m.cov[from * 6 + a] : 0.f;
            }
            if (cov_ok) cov_ok[to] = (have && m.cov_ok) ? m.cov_ok[from] : 0;
        }
    }
}

__global__ void write_i64_kernel(const unsigned long long* src, int64_t* dst) {
    if (threadIdx.x == 0 && blockIdx.x == 0) *dst = (int64_t)*src;
}

__global__ void __launch_bounds__(256) voxel_keys_kernel(const float* __restrict__ xyz, int64_t n, int stride, float v,
                                                          unsigned long long* __restrict__ keys) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float* p = xyz + i * stride;
    int k[3];
    keys[i] = voxel_index(p[0], p[1], p[2], v, k) ? pack_key(k[0], k[1], k[2]) : KEY_EMPTY;
}

// ---- rehash: move the live voxels into a clean table (drops dead keys) --------------------------------------
// pass 1 copies every live bucket into a compact temporary; pass 2 re-inserts them after the table was cleared
__global__ void __launch_bounds__(256) rehash_gather_kernel(MapView m, unsigned long long* __restrict__ keys,
                                                             uint32_t* __restrict__ counts, float4* __restrict__ pts,
                                                             float* __restrict__ cov6, uint8_t* __restrict__ cov_ok,
                                                             unsigned long long* n_out) {
    const uint32_t s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= m.slots) return;
    const Entry e = m.table[s];
    if (e.key == KEY_EMPTY) return;
    float4* bucket = m.points + (size_t)s * m.cap;
    if (e.count > 0) {
        const unsigned long long r = atomicAdd(n_out, 1ull);
        keys[r] = e.key;
        counts[r] = e.count;
        for (uint32_t j = 0; j < e.count; ++j) {
            const size_t from = (size_t)s * m.cap + j, to = (size_t)r * m.cap + j;
            pts[to] = bucket[j];
            if (m.cov) {
                for (int a = 0; a < 6; ++a) cov6[to * 6 + a] = m.cov[from * 6 + a];
                cov_ok[to] = m.cov_ok[from];
            }
        }
    }
    for (uint32_t j = 0; j < e.count; ++j) m.ids[(size_t)s * m.cap + j] = NO_ID;
    Entry z;
    z.key = KEY_EMPTY; z.count = 0; z.pad = 0;
    m.table[s] = z;
}

__global__ void __launch_bounds__(256) rehash_scatter_kernel(MapView m, const unsigned long long* __restrict__ keys,
                                                              const uint32_t* __restrict__ counts,
                                                              const float4* __restrict__ pts, const float* __restrict__ cov6,
                                                              const uint8_t* __restrict__ cov_ok,
                                                              const unsigned long long* n_live) {
    const unsigned long long r = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= *n_live) return;
    const unsigned long long key = keys[r];
    uint32_t s = hash_key(key) & m.mask;
    for (uint32_t probes = 0; probes < m.slots; ++probes) {
        if (atomicCAS(&m.table[s].key, KEY_EMPTY, key) == KEY_EMPTY) {
            atomicMax(&m.table[hash_key(key) & m.mask].pad, probes + 1u);
            break;
        }
        s = (s + 1) & m.mask;
    }
    const uint32_t cnt = counts[r];
    for (uint32_t j = 0; j < cnt; ++j) {
        const size_t to = (size_t)s * m.cap + j, from = (size_t)r * m.cap + j;
        m.points[to] = pts[from];
        m.ids[to] = __float_as_uint(pts[from].w);
        if (m.cov) {
            for (int a = 0; a < 6; ++a) m.cov[to * 6 + a] = cov6[from * 6 + a];
            m.cov_ok[to] = cov_ok[from];
        }
    }
    m.table[s].count = cnt;
    if (r == 0) m.ctr->n_keys = *n_live;
}

}  // namespace far

// =============================================================================================================
extern "C" {

const char* far_strerror(int status) {
    switch (status) {
        case FAR_OK: return "ok";
        case FAR_ERR_ARG: return "invalid argument";
        case FAR_ERR_CUDA: return "CUDA runtime error";
        case FAR_ERR_FULL: return "voxel table full";
        case FAR_ERR_RANGE: return "point id counter out of range";
        case FAR_ERR_DEGENERATE: return "degenerate registration (too few inliers or H not positive definite)";
        default: return "unknown status";
    }
}

const char* far_last_cuda_error(void) { return far::g_cuda_err; }

int far_map_create(far_map_t** out, const far_map_config_t* cfg) {
    if (!out || !cfg) return FAR_ERR_ARG;
    *out = nullptr;
    far_map_config_t c = *cfg;
    if (!(c.voxel_size > 0.f) || c.cap < 1 || c.cap > 64 || c.max_voxels < 1) return FAR_ERR_ARG;
    if (c.max_load == 0.f) c.max_load = 0.5f;
    if (!(c.max_load > 0.f && c.max_load <= 0.9f)) return FAR_ERR_ARG;
    if (c.k_cov == 0) c.k_cov = 10;
    if (c.k_cov < 1 || c.k_cov > 32) return FAR_ERR_ARG;
    if (c.cov_eps == 0.0) c.cov_eps = 1e-3;
    if (c.max_batch == 0) c.max_batch = 1 << 20;
    if (c.max_batch < 1 || c.max_batch > (1ll << 30)) return FAR_ERR_ARG;
    uint64_t slots = 16;
    const double want = (double)c.max_voxels / (double)c.max_load;
    while ((double)slots < want) slots <<= 1;
    if (slots * (uint64_t)c.cap >= (1ull << 32)) return FAR_ERR_ARG;   // refs (slot*cap+pos) are 32-bit

    far_map* m = new (std::nothrow) far_map();
    if (!m) return FAR_ERR_ARG;
    memset(m, 0, sizeof(*m));
    m->cfg = c;
    m->max_batch = c.max_batch;
    m->next_id = 0;
    FAR_CUDA(cudaGetDevice(&m->device));
    FAR_CUDA(cudaDeviceGetAttribute(&m->sm_count, cudaDevAttrMultiProcessorCount, m->device));
    MapView& v = m->view;
    v.slots = (uint32_t)slots;
    v.mask = (uint32_t)slots - 1;
    v.cap = c.cap;
    v.k_cov = c.k_cov;
    v.voxel = c.voxel_size;
    v.cov_eps = c.cov_eps;
    v.max_keys = (unsigned long long)c.max_voxels;
    const size_t npts = (size_t)slots * c.cap;
    cudaError_t e = cudaSuccess;
    auto alloc = [&](void** p, size_t bytes) { if (e == cudaSuccess) e = cudaMalloc(p, bytes); };
    alloc((void**)&v.table, slots * sizeof(Entry));
    alloc((void**)&v.points, npts * sizeof(float4));
    alloc((void**)&v.ids, npts * sizeof(uint32_t));
    if (c.with_cov) {
        alloc((void**)&v.cov, npts * 6 * sizeof(float));
        alloc((void**)&v.cov_ok, npts);
    }
    alloc((void**)&v.ctr, sizeof(Counters) + 8 * sizeof(unsigned long long));
    alloc((void**)&m->d_touched, (size_t)c.max_batch * 4);
    alloc((void**)&m->d_cov_list, (size_t)c.max_batch * 4);
    if (e != cudaSuccess) {
        far::set_cuda_error(e, "cudaMalloc in far_map_create");
        far_map_destroy(m);
        return FAR_ERR_CUDA;
    }
    // empty table: every key = ~0, count = 0; every id word = FAR_NO_ID
    FAR_CUDA(cudaMemset(v.ids, 0xFF, npts * sizeof(uint32_t)));
    FAR_LAUNCH(table_init_kernel, grid_for((int64_t)slots, 256), 256, 0, 0, v.table, v.slots);
    FAR_CUDA(cudaGetLastError());
    FAR_CUDA(cudaMemset(v.ctr, 0, sizeof(Counters) + 8 * sizeof(unsigned long long)));
    if (v.cov_ok) FAR_CUDA(cudaMemset(v.cov_ok, 0, npts));
    {
        const int rc = gicp_setup(m);
        if (rc != FAR_OK) { far_map_destroy(m); return rc; }
    }
    FAR_CUDA(cudaDeviceSynchronize());
    *out = m;
    return FAR_OK;
}

int far_map_destroy(far_map_t* m) {
    if (!m) return FAR_OK;
    cudaFree(m->view.table); cudaFree(m->view.points); cudaFree(m->view.ids); cudaFree(m->view.cov); cudaFree(m->view.cov_ok);
    cudaFree(m->view.ctr); cudaFree(m->d_touched); cudaFree(m->d_cov_list);
    cudaFree(m->d_gicp_partials);
    delete m;
    return FAR_OK;
}

int far_map_clear(far_map_t* m, void* stream) {
    if (!m) return FAR_ERR_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    FAR_LAUNCH(clear_kernel, grid_for(m->view.slots, 256), 256, 0, st, m->view);
    FAR_CUDA(cudaGetLastError());
    FAR_CUDA(cudaMemsetAsync(m->view.ctr, 0, sizeof(Counters), st));
    m->next_id = 0;
    return FAR_OK;
}

static int insert_impl(far_map_t* m, const float* d_xyz, int64_t n, int stride, int pose_mode, const far_pose_t* hpose,
                       const far_pose_t* d_pose, int compute_cov, far_insert_stats_t* d_stats, void* stream,
                       Asmd asmd = Asmd{nullptr, 1.0, 0}) {
    if (!m || (!d_xyz && n > 0) || n < 0 || (stride != 3 && stride != 4)) return FAR_ERR_ARG;
    if (compute_cov && !m->view.cov) return FAR_ERR_ARG;
    if (m->next_id + (uint64_t)n > 0xFFFFFFFFull) return FAR_ERR_RANGE;
    cudaStream_t st = (cudaStream_t)stream;
    Pose hp;
    memset(&hp, 0, sizeof(hp));
    if (pose_mode == 1) memcpy(&hp, hpose, sizeof(hp));
    Counters* ctr = m->view.ctr;
    // zero the touched counter, the covariance queue and the per-call statistics (contiguous: one call)
    FAR_CUDA(cudaMemsetAsync(&ctr->n_touched, 0, 2 * sizeof(unsigned int) + 4 * sizeof(unsigned long long), st));
    const bool cov_by_list = compute_cov && n <= m->max_batch;
    const uint32_t call_first_id = (uint32_t)m->next_id;
    const int commit_grid = m->sm_count * 8;
    for (int64_t off = 0; off < n; off += m->max_batch) {
        const int64_t nc = (n - off < m->max_batch) ? n - off : m->max_batch;
        const uint32_t first_id = (uint32_t)(m->next_id + (uint64_t)off);
        const float* xyz = d_xyz + off * stride;
        if (off > 0) FAR_CUDA(cudaMemsetAsync(&ctr->n_touched, 0, sizeof(unsigned int), st));
        FAR_LAUNCH(insert_claim_chain_kernel, grid_for(nc, 256), 256, 0, st, m->view, xyz, nc, stride, pose_mode, hp,
                                                                      (const Pose*)d_pose, first_id, m->d_touched, asmd);
        FAR_LAUNCH(insert_commit_kernel, commit_grid, 256, 0, st, m->view, xyz, stride, pose_mode, hp, (const Pose*)d_pose,
                                                           first_id, m->d_touched, cov_by_list ? m->d_cov_list : nullptr,
                                                           m->max_batch);
        FAR_CUDA(cudaGetLastError());
    }
    m->next_id += (uint64_t)n;
    if (compute_cov && n > 0) {
        // "we recompute the covariances of the added points" -- against the map AFTER the insert
        int rc = cov_by_list ? launch_knn_cov_refs(m, m->d_cov_list, &ctr->n_cov, n, st)
                             : launch_knn_cov_new_ids(m, call_first_id, st);
        if (rc != FAR_OK) return rc;
    }
    if (d_stats) {
        FAR_LAUNCH(insert_stats_kernel, 1, 32, 0, st, m->view, n, d_stats);
        FAR_CUDA(cudaGetLastError());
    }
    return FAR_OK;
}

int far_map_insert(far_map_t* m, const float* d_xyz, int64_t n, int stride, const far_pose_t* pose, int compute_cov,
                   far_insert_stats_t* d_stats, void* stream) {
    return insert_impl(m, d_xyz, n, stride, pose ? 1 : 0, pose, nullptr, compute_cov, d_stats, stream);
}

int far_map_insert_dev(far_map_t* m, const float* d_xyz, int64_t n, int stride, const far_pose_t* d_pose,
                       int compute_cov, far_insert_stats_t* d_stats, void* stream) {
    if (!d_pose) return FAR_ERR_ARG;
    return insert_impl(m, d_xyz, n, stride, 2, nullptr, d_pose, compute_cov, d_stats, stream);
}

int far_map_insert_asmd(far_map_t* m, const float* d_xyz, int64_t n, int stride, const far_pose_t* pose,
                        const double* d_n_close, double d_max, int compute_cov, far_insert_stats_t* d_stats, void* stream) {
    if (!d_n_close || !(d_max > 0.0)) return FAR_ERR_ARG;
    return insert_impl(m, d_xyz, n, stride, pose ? 1 : 0, pose, nullptr, compute_cov, d_stats, stream, Asmd{d_n_close, d_max, 1});
}

int far_map_insert_asmd_dev(far_map_t* m, const float* d_xyz, int64_t n, int stride, const far_pose_t* d_pose,
                            const double* d_n_close, double d_max, int compute_cov, far_insert_stats_t* d_stats,
                            void* stream) {
    if (!d_pose || !d_n_close || !(d_max > 0.0)) return FAR_ERR_ARG;
    return insert_impl(m, d_xyz, n, stride, 2, nullptr, d_pose, compute_cov, d_stats, stream, Asmd{d_n_close, d_max, 1});
}

// PAPER.md:109 "the average amount of points per voxel in a close range of the current scan" (R17)
int far_asmd_density(const far_map_t* local, const double center[3], double r_close, double* d_out, void* stream) {
    if (!local || !center || !d_out || !(r_close >= 0.0)) return FAR_ERR_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    unsigned long long* acc = reinterpret_cast<unsigned long long*>(local->view.ctr + 1) + 4;   // 2 words of the tail
    FAR_CUDA(cudaMemsetAsync(acc, 0, 2 * sizeof(unsigned long long), st));
    FAR_LAUNCH(asmd_density_kernel, grid_for(local->view.slots, 256), 256, 0, st, local->view, center[0], center[1], center[2],
                                                                        r_close * r_close, acc);
    FAR_LAUNCH(asmd_density_out_kernel, 1, 32, 0, st, local->view, acc, d_out);
    FAR_CUDA(cudaGetLastError());
    return FAR_OK;
}

static int prune_impl(far_map_t* m, const double* c, const far_pose_t* d_pose, double radius, far_prune_stats_t* d_stats,
                      void* stream) {
    if (!m || (!c && !d_pose)) return FAR_ERR_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    const double r2 = radius * radius;
    FAR_LAUNCH(prune_kernel, grid_for(m->view.slots, 256), 256, 0, st, m->view, c ? c[0] : 0.0, c ? c[1] : 0.0, c ? c[2] : 0.0,
                                                                (const Pose*)d_pose, r2, d_stats);
    FAR_CUDA(cudaGetLastError());
    return FAR_OK;
}

int far_map_prune(far_map_t* m, const double center[3], double radius, far_prune_stats_t* d_stats, void* stream) {
    if (!center) return FAR_ERR_ARG;
    return prune_impl(m, center, nullptr, radius, d_stats, stream);
}

int far_map_prune_dev(far_map_t* m, const far_pose_t* d_pose, double radius, far_prune_stats_t* d_stats, void* stream) {
    if (!d_pose) return FAR_ERR_ARG;
    return prune_impl(m, nullptr, d_pose, radius, d_stats, stream);
}

int far_map_stats(far_map_t* m, far_map_stats_t* d_stats, void* stream) {
    if (!m || !d_stats) return FAR_ERR_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    unsigned long long* acc = reinterpret_cast<unsigned long long*>(m->view.ctr + 1);
    FAR_LAUNCH(stats_kernel, grid_for(m->view.slots, 256), 256, 0, st, m->view, acc);
    FAR_LAUNCH(stats_out_kernel, 1, 32, 0, st, m->view, acc, m->next_id, d_stats);
    FAR_CUDA(cudaGetLastError());
    return FAR_OK;
}

int far_map_export(far_map_t* m, uint64_t* d_keys, int32_t* d_counts, float* d_points4, float* d_cov6,
                   uint8_t* d_cov_valid, int64_t max_out, int64_t* d_n_voxels, void* stream) {
    if (!m || !d_keys || !d_counts || !d_n_voxels || max_out < 0) return FAR_ERR_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    unsigned long long* acc = reinterpret_cast<unsigned long long*>(m->view.ctr + 1) + 3;
    FAR_CUDA(cudaMemsetAsync(acc, 0, sizeof(unsigned long long), st));
    FAR_LAUNCH(export_kernel, grid_for(m->view.slots, 256), 256, 0, st, m->view, (unsigned long long*)d_keys, d_counts,
                                                                 (float4*)d_points4, d_cov6, d_cov_valid, max_out, acc);
    FAR_LAUNCH(write_i64_kernel, 1, 32, 0, st, acc, d_n_voxels);
    FAR_CUDA(cudaGetLastError());
    return FAR_OK;
}

int far_voxel_keys(const float* d_xyz, int64_t n, int stride, float voxel, uint64_t* d_keys, void* stream) {
    if ((!d_xyz && n > 0) || n < 0 || (stride != 3 && stride != 4) || !(voxel > 0.f) || (!d_keys && n > 0)) return FAR_ERR_ARG;
    if (n == 0) return FAR_OK;
    FAR_LAUNCH(voxel_keys_kernel, grid_for(n, 256), 256, 0, (cudaStream_t)stream, d_xyz, n, stride, voxel,
                                                                          (unsigned long long*)d_keys);
    FAR_CUDA(cudaGetLastError());
    return FAR_OK;
}

// Maintenance call (not on the per-frame hot path): allocates a compact temporary for the live voxels,
// synchronises the stream once to learn their number, and frees the temporary before returning.
int far_map_rehash(far_map_t* m, void* stream) {
    if (!m) return FAR_ERR_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    far_map_stats_t hs;
    far_map_stats_t* d_hs = nullptr;
    FAR_CUDA(cudaMalloc((void**)&d_hs, sizeof(hs)));
    int rc = far_map_stats(m, d_hs, stream);
    if (rc != FAR_OK) { cudaFree(d_hs); return rc; }
    FAR_CUDA(cudaMemcpyAsync(&hs, d_hs, sizeof(hs), cudaMemcpyDeviceToHost, st));
    FAR_CUDA(cudaStreamSynchronize(st));
    cudaFree(d_hs);
    const size_t nv = (size_t)hs.n_voxels, cap = (size_t)m->view.cap;
    unsigned long long *t_keys = nullptr, *t_n = nullptr;
    uint32_t* t_counts = nullptr;
    float4* t_pts = nullptr;
    float* t_cov = nullptr;
    uint8_t* t_ok = nullptr;
    cudaError_t e = cudaMalloc((void**)&t_keys, (nv + 1) * 8);
    if (e == cudaSuccess) e = cudaMalloc((void**)&t_counts, (nv + 1) * 4);
    if (e == cudaSuccess) e = cudaMalloc((void**)&t_pts, (nv * cap + 1) * sizeof(float4));
    if (e == cudaSuccess) e = cudaMalloc((void**)&t_n, 8);
    if (e == cudaSuccess && m->view.cov) e = cudaMalloc((void**)&t_cov, (nv * cap + 1) * 6 * sizeof(float));
    if (e == cudaSuccess && m->view.cov) e = cudaMalloc((void**)&t_ok, nv * cap + 1);
    if (e == cudaSuccess) e = cudaMemsetAsync(t_n, 0, 8, st);
    if (e == cudaSuccess) {
        FAR_LAUNCH(rehash_gather_kernel, grid_for(m->view.slots, 256), 256, 0, st, m->view, t_keys, t_counts, t_pts, t_cov, t_ok, t_n);
        if (nv > 0)
            FAR_LAUNCH(rehash_scatter_kernel, grid_for((int64_t)nv, 256), 256, 0, st, m->view, t_keys, t_counts, t_pts, t_cov, t_ok, t_n);
        else
            e = cudaMemsetAsync(&m->view.ctr->n_keys, 0, 8, st);
        if (e == cudaSuccess) e = cudaGetLastError();
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    }
    cudaFree(t_keys); cudaFree(t_counts); cudaFree(t_pts); cudaFree(t_n); cudaFree(t_cov); cudaFree(t_ok);
    if (e != cudaSuccess) { far::set_cuda_error(e, "far_map_rehash"); return FAR_ERR_CUDA; }
    return FAR_OK;
}

}  // extern "C"

// =============================================================================================================
// launch accounting / per-kernel timing (tracing facility) and map snapshots (checkpoint / restore)
#include <atomic>
#include <map>
#include <mutex>
#include <string>
#include <vector>

namespace far {

static std::atomic<long long> g_launches{0};
static std::atomic<int> g_prof{0};
static std::mutex g_prof_mu;
struct ProfRec { const char* name; cudaEvent_t a, b; };
static std::vector<ProfRec> g_recs;

LaunchScope::LaunchScope(const char* name, cudaStream_t st) : rec_(-1), st_(st) {
    g_launches.fetch_add(1, std::memory_order_relaxed);
    if (g_prof.load(std::memory_order_relaxed)) {
        ProfRec r;
        r.name = name;
        if (cudaEventCreate(&r.a) == cudaSuccess && cudaEventCreate(&r.b) == cudaSuccess) {
            cudaEventRecord(r.a, st);
            std::lock_guard<std::mutex> lk(g_prof_mu);
            g_recs.push_back(r);
            rec_ = (int)g_recs.size() - 1;
        }
    }
}

LaunchScope::~LaunchScope() {
    if (rec_ >= 0) {
        std::lock_guard<std::mutex> lk(g_prof_mu);
        cudaEventRecord(g_recs[rec_].b, st_);
    }
}

}  // namespace far

struct far_snapshot {
    void *table, *points, *ids, *cov, *cov_ok, *ctr;
    size_t b_table, b_points, b_ids, b_cov, b_ok;
    uint64_t next_id;
};

extern "C" {

long long far_launch_count(void) { return far::g_launches.load(); }

void far_profile_enable(int on) { far::g_prof.store(on ? 1 : 0); }

// Synchronises the device, sums the recorded durations per kernel name and clears the records.
// Writes up to max_entries rows: names[i] (borrowed static strings), total_ms[i], launches[i]; returns the row count.
int far_profile_collect(const char** names, double* total_ms, long long* launches, int max_entries) {
    cudaDeviceSynchronize();
    std::lock_guard<std::mutex> lk(far::g_prof_mu);
    std::map<std::string, std::pair<double, long long>> acc;
    std::map<std::string, const char*> ptr;
    for (auto& r : far::g_recs) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, r.a, r.b) == cudaSuccess) {
            auto& e = acc[r.name];
            e.first += ms;
            e.second += 1;
            ptr[r.name] = r.name;
        }
        cudaEventDestroy(r.a);
        cudaEventDestroy(r.b);
    }
    far::g_recs.clear();
    int i = 0;
    for (auto& kv : acc) {
        if (i >= max_entries) break;
        if (names) names[i] = ptr[kv.first];
        if (total_ms) total_ms[i] = kv.second.first;
        if (launches) launches[i] = kv.second.second;
        ++i;
    }
    return i;
}

int far_map_snapshot_destroy(far_snapshot_t* s) {
    if (!s) return FAR_OK;
    cudaFree(s->table); cudaFree(s->points); cudaFree(s->ids); cudaFree(s->cov); cudaFree(s->cov_ok); cudaFree(s->ctr);
    delete s;
    return FAR_OK;
}

int far_map_snapshot_create(far_map_t* m, far_snapshot_t** out, void* stream) {
    if (!m || !out) return FAR_ERR_ARG;
    *out = nullptr;
    cudaStream_t st = (cudaStream_t)stream;
    far_snapshot* s = new (std::nothrow) far_snapshot();
    if (!s) return FAR_ERR_ARG;
    memset(s, 0, sizeof(*s));
    const size_t npts = (size_t)m->view.slots * m->view.cap;
    s->b_table = (size_t)m->view.slots * sizeof(Entry);
    s->b_points = npts * sizeof(float4);
    s->b_ids = npts * sizeof(uint32_t);
    s->b_cov = m->view.cov ? npts * 6 * sizeof(float) : 0;
    s->b_ok = m->view.cov_ok ? npts : 0;
    s->next_id = m->next_id;
    cudaError_t e = cudaMalloc(&s->table, s->b_table);
    if (e == cudaSuccess) e = cudaMalloc(&s->points, s->b_points);
    if (e == cudaSuccess) e = cudaMalloc(&s->ids, s->b_ids);
    if (e == cudaSuccess && s->b_cov) e = cudaMalloc(&s->cov, s->b_cov);
    if (e == cudaSuccess && s->b_ok) e = cudaMalloc(&s->cov_ok, s->b_ok);
    if (e == cudaSuccess) e = cudaMalloc(&s->ctr, sizeof(Counters));
    if (e == cudaSuccess) e = cudaMemcpyAsync(s->table, m->view.table, s->b_table, cudaMemcpyDeviceToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(s->points, m->view.points, s->b_points, cudaMemcpyDeviceToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(s->ids, m->view.ids, s->b_ids, cudaMemcpyDeviceToDevice, st);
    if (e == cudaSuccess && s->b_cov) e = cudaMemcpyAsync(s->cov, m->view.cov, s->b_cov, cudaMemcpyDeviceToDevice, st);
    if (e == cudaSuccess && s->b_ok) e = cudaMemcpyAsync(s->cov_ok, m->view.cov_ok, s->b_ok, cudaMemcpyDeviceToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(s->ctr, m->view.ctr, sizeof(Counters), cudaMemcpyDeviceToDevice, st);
    if (e != cudaSuccess) {
        far::set_cuda_error(e, "far_map_snapshot_create");
        far_map_snapshot_destroy(s);
        return FAR_ERR_CUDA;
    }
    *out = s;
    return FAR_OK;
}

int far_map_snapshot_restore(far_map_t* m, const far_snapshot_t* s, void* stream) {
    if (!m || !s) return FAR_ERR_ARG;
    const size_t npts = (size_t)m->view.slots * m->view.cap;
    if (s->b_table != (size_t)m->view.slots * sizeof(Entry) || s->b_points != npts * sizeof(float4)) return FAR_ERR_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    FAR_CUDA(cudaMemcpyAsync(m->view.table, s->table, s->b_table, cudaMemcpyDeviceToDevice, st));
    FAR_CUDA(cudaMemcpyAsync(m->view.points, s->points, s->b_points, cudaMemcpyDeviceToDevice, st));
    FAR_CUDA(cudaMemcpyAsync(m->view.ids, s->ids, s->b_ids, cudaMemcpyDeviceToDevice, st));
    if (s->b_cov && m->view.cov) FAR_CUDA(cudaMemcpyAsync(m->view.cov, s->cov, s->b_cov, cudaMemcpyDeviceToDevice, st));
    if (s->b_ok && m->view.cov_ok) FAR_CUDA(cudaMemcpyAsync(m->view.cov_ok, s->cov_ok, s->b_ok, cudaMemcpyDeviceToDevice, st));
    FAR_CUDA(cudaMemcpyAsync(m->view.ctr, s->ctr, sizeof(Counters), cudaMemcpyDeviceToDevice, st));
    m->next_id = s->next_id;
    return FAR_OK;
}

}  // extern "C"
