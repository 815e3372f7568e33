// far_common.cuh -- device-side building blocks shared by the far_* kernels (sm_100a).
//
// Layout of the voxel hashmap in HBM ("cuVoxelMap"; re-designed for B200):
//   table   : Entry[slots]              16 B per slot {u64 key, u32 bucket, u32 count | reach << 8}; one LDG.128 yields the
//                                       key, where its points live AND how many there are, so a lookup is two dependent
//                                       memory levels (entry -> points), not three.
//   shadow  : Entry[slots]              second table of the same size, empty between calls: the target of the in-place
//                                       rehash that drops the keys of pruned voxels (rehash_*_kernel in far_map.cu)
//   points  : float4[max_voxels * cap]  DENSE bucket pool (Fig. 3: points stored apart from the key table);
//                                       bucket b = points[b*cap .. b*cap+cap); .w = id bits; positions >= count never read.
//                                       Buckets come from a bump allocator and a free list refilled by pruning, so V live
//                                       voxels occupy V * cap * 16 B contiguous-ish bytes whatever the table size.
//   ids     : u32[max_voxels * cap]     the id of stored point j of bucket b at ids[b*cap + j], FAR_NO_ID if the position
//                                       is free: the working storage of the deterministic insert (its atomicMin chain
//                                       touches 80 contiguous bytes per voxel at cap 20)
//   cov     : float[max_voxels*cap*6]   (optional) regularised covariance of each stored point (Eq. 1)
//   cov_ok  : u8[max_voxels * cap]      (optional) 1 if that covariance is valid (>= k neighbours)
//   free    : u32[max_voxels]           stack of bucket indices returned by far_map_prune
//   occ     : u32[slots / 32]           one bit per table slot "holds a key" (set when a key is claimed, recomputed by the
//                                       rehash): L2-resident filter in front of the table for the NN sweep
// A pruned voxel gives its bucket back at once; its key stays in the table with bucket = NO_BUCKET ("dead key": absent for
// every query, re-usable by an insert) until the number of dead keys passes a device-side threshold, at which point the
// prune call's rehash kernel rebuilds the 16-byte entries into `shadow` and copies them back -- no allocation, no host sync.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/far.h"

namespace far {

constexpr unsigned long long KEY_EMPTY = ~0ull;
constexpr uint32_t NO_ID = 0xFFFFFFFFu;
constexpr uint32_t NO_SLOT = 0xFFFFFFFFu;
constexpr uint32_t NO_BUCKET = 0xFFFFFFFFu;        // key present, no points: pruned (dead key) or the pool was exhausted
constexpr uint32_t BUCKET_PENDING = 0xFFFFFFFEu;   // the bucket word of every EMPTY slot; on a claimed key: the claimer (or
                                                   // the thread that revives a dead key) is allocating the bucket right now
constexpr int KEY_BIAS = 1 << 20;
constexpr unsigned FULL = 0xFFFFFFFFu;
constexpr uint32_t TOUCHED_SUBS = 32;             // sub-lists of the insert's touched list (far_map.cu)

struct __align__(16) Entry {
    unsigned long long key;
    uint32_t bucket;   // index into the dense pool, NO_BUCKET, or BUCKET_PENDING (only while an insert kernel runs)
    uint32_t cr;       // bits 0..7: number of stored points; bits 8..31: reach of this HOME slot = the largest
                       // displacement of any key whose home slot this is (see find_voxel)
};

// device counters of one map (all zeroed at create / clear)
struct Counters {
    unsigned long long next_id;       // id of the next offered point (device-resident: no per-call kernel argument)
    unsigned long long call_first_id; // first id of the insert call whose last chunk was committed most recently
    unsigned int n_keys;              // claimed keys (live + dead)
    unsigned int n_dead;              // keys in the table that own no bucket: voxels pruned since the last rehash and not opened
                                      // again since, plus keys claimed when the bucket pool was exhausted
    unsigned int bump;                // buckets ever taken from the fresh end of the pool
    int n_free;                       // entries on the free list
    unsigned int n_alloc;             // buckets handed out by the running insert kernel: the first n_free of them come off the
                                      // free list, the rest from the fresh end; folded into n_free / bump by the commit epilogue
    unsigned int full_flag;           // sticky until buckets are freed: a point was dropped (pool or table exhausted)
    unsigned int rehash_flag;         // written by prune's epilogue: the rehash kernel that follows does its work (and clears it)
    unsigned int rehash_moved;        // entries moved by the running rehash
    unsigned int n_rehash;            // rehashes done since create / clear
    unsigned int ticket[6];           // last-block-done tickets: 0 insert commit, 1 prune, 2 clear, 3 renumber, 4 rehash
    unsigned int rehash_barrier;      // arrivals at the grid-wide barrier between the two passes of the rehash
    unsigned int n_tasks;             // length of the covariance queue the last insert call left for knn_cov_refs_kernel
    unsigned int min_id;              // far_map_renumber: smallest live id
    unsigned int n_cov;               // accepted points queued for covariance by the running insert call
    unsigned long long st_accepted, st_new_voxels, st_dropped_full, st_invalid;   // per-call statistics
    unsigned long long pr_vox_removed, pr_pts_removed, pr_vox_left, pr_pts_left;  // per-prune statistics
    unsigned long long scratch[8];    // stats / export / ASMD accumulators
};

// written by the device into pinned, mapped HOST memory: lets later host calls report conditions without a sync
struct Mailbox {
    volatile uint32_t full;             // mirrors Counters::full_flag
    volatile uint32_t renumber_seq;     // 2 x far_map_renumber passes completed; odd while a pass writes the two words below
    volatile unsigned long long next_id_after_renumber;
    volatile unsigned long long offered_at_renumber;   // host-side offered-points counter the pass was enqueued at
};

// device view of a map, passed by value to kernels
struct MapView {
    Entry* table;
    Entry* shadow;
    float4* points;
    uint32_t* ids;
    float* cov;          // nullable
    uint8_t* cov_ok;     // nullable
    uint32_t* free_list;
    uint32_t* occ;       // [slots / 32] one bit per table slot: the slot holds a key.  8 MB for the 2^26-slot table of a 20 M-voxel map:
                         // it stays in the 126 MB L2, so a lookup whose home slot is empty costs no DRAM access at all (find_voxel<true>)
    Counters* ctr;
    Mailbox* mail;       // device pointer to the mapped host mailbox
    uint32_t* touched_cnt;   // [TOUCHED_SUBS][32]: lengths of the sub-lists of the insert's touched list, one 128-byte line each
    uint32_t touched_sub_cap;   // capacity of one sub-list
    uint32_t mask;       // slots - 1
    uint32_t slots;
    uint32_t max_buckets;
    uint32_t key_limit;  // new keys are refused beyond this many claimed slots (probe lengths stay bounded)
    int cap;
    int k_cov;
    float voxel;
    double cov_eps;
};

struct Pose {
    double R[9];
    double t[3];
};

__device__ __forceinline__ uint32_t entry_count(uint32_t cr) { return cr & 0xFFu; }
__device__ __forceinline__ uint32_t entry_reach(uint32_t cr) { return cr >> 8; }

// true in exactly one block of the grid: the one whose thread 0 takes the last ticket, after every other block has
// passed this point (its earlier writes are fenced).  All threads of the block must call; the ticket re-arms itself.
__device__ __forceinline__ bool last_block_done(unsigned int* ticket) {
    __shared__ bool s_last;
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) {
        const bool last = atomicAdd(ticket, 1u) == gridDim.x - 1;
        if (last) { *ticket = 0u; __threadfence(); }
        s_last = last;
    }
    __syncthreads();
    return s_last;
}

// ---- A1: voxel key (R1).  One IEEE fp32 division, floor, 21-bit biased pack. -------------
__device__ __forceinline__ bool voxel_index(float x, float y, float z, float v, int k[3]) {
    if (!(isfinite(x) && isfinite(y) && isfinite(z))) return false;
    const float fx = floorf(__fdiv_rn(x, v));
    const float fy = floorf(__fdiv_rn(y, v));
    const float fz = floorf(__fdiv_rn(z, v));
    const bool ok = (fx >= -1048576.0f && fx < 1048576.0f) && (fy >= -1048576.0f && fy < 1048576.0f) &&
                    (fz >= -1048576.0f && fz < 1048576.0f);
    if (!ok) return false;
    k[0] = (int)fx; k[1] = (int)fy; k[2] = (int)fz;
    return true;
}

__device__ __forceinline__ unsigned long long pack_key(int kx, int ky, int kz) {
    return ((unsigned long long)(uint32_t)(kx + KEY_BIAS) << 42) | ((unsigned long long)(uint32_t)(ky + KEY_BIAS) << 21) |
           (unsigned long long)(uint32_t)(kz + KEY_BIAS);
}

__device__ __forceinline__ void unpack_key(unsigned long long key, int k[3]) {
    k[0] = (int)((key >> 42) & 0x1FFFFF) - KEY_BIAS;
    k[1] = (int)((key >> 21) & 0x1FFFFF) - KEY_BIAS;
    k[2] = (int)(key & 0x1FFFFF) - KEY_BIAS;
}

__device__ __forceinline__ bool index_in_range(int k) { return k >= -KEY_BIAS && k < KEY_BIAS; }

// Spatial hash of the packed key (PAPER.md:62 cites Niessner et al. for its hash; slot placement is not
// observable, so the mixing function is a free choice): 64-bit finaliser-style avalanche.
__device__ __forceinline__ uint32_t hash_key(unsigned long long k) {
    k ^= k >> 33;
    k *= 0xff51afd7ed558ccdULL;
    k ^= k >> 33;
    k *= 0xc4ceb9fe1a85ec53ULL;
    k ^= k >> 33;
    return (uint32_t)k;
}

// ---- A4: rigid transform (R4): ((R0 x + R1 y) + R2 z) + t, every operation one rounded binary64 op --------
__device__ __forceinline__ void transform_point(const Pose& T, float sx, float sy, float sz, float out[3]) {
    const double x = (double)sx, y = (double)sy, z = (double)sz;
#pragma unroll
    for (int r = 0; r < 3; ++r) {
        double acc = __dadd_rn(__dmul_rn(T.R[3 * r + 0], x), __dmul_rn(T.R[3 * r + 1], y));
        acc = __dadd_rn(acc, __dmul_rn(T.R[3 * r + 2], z));
        acc = __dadd_rn(acc, T.t[r]);
        out[r] = __double2float_rn(acc);
    }
}

// ---- A6: squared distance (R6): exact differences, (dx^2 + dy^2) + dz^2 in rounded binary64 ops ---------
__device__ __forceinline__ double dist2(float qx, float qy, float qz, float px, float py, float pz) {
    const double dx = (double)qx - (double)px;
    const double dy = (double)qy - (double)py;
    const double dz = (double)qz - (double)pz;
    return __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
}

__device__ __forceinline__ Entry load_entry(const Entry* table, uint32_t s) {
    const uint4 raw = __ldg(reinterpret_cast<const uint4*>(table + s));
    Entry e;
    e.key = ((unsigned long long)raw.y << 32) | raw.x;
    e.bucket = raw.z;
    e.cr = raw.w;
    return e;
}

// read-only lookup: bucket of `key` and its count, or NO_BUCKET / count = 0 if absent or dead.  Linear probing, step 1
// (PAPER.md:62).  The upper 24 bits of the entry at a key's HOME slot h hold `reach` = the largest displacement of any key
// whose home is h (raised when a displaced key is claimed, recomputed by every rehash).  A lookup therefore examines the
// slots h .. h + reach(h) only: a voxel that is not in the map -- 11 of the 27 neighbours of a typical query -- is usually
// dismissed by the one home-entry load instead of a walk to the next empty slot, and the warp no longer waits for the
// longest of 27 such walks.  An EMPTY home slot means no key has that home (keys are only ever removed by a rebuild).
// USE_OCC: the home slot's bit of the occupancy bitmap is looked at first (an L2 hit) and an empty home slot is settled
// without touching the table -- for throughput-bound sweeps over maps far larger than L2 (nn_kernel at C5: 25 of the 27
// neighbours of a query are absent at v = 0.25 and three quarters of them have an empty home slot); the latency-bound
// frame kernels go straight to the entry (the bitmap would be one more dependent level for the voxels that exist).
template <bool USE_OCC = false>
__device__ __forceinline__ uint32_t find_voxel(const MapView& m, unsigned long long key, uint32_t& count) {
    const uint32_t h = hash_key(key) & m.mask;
    count = 0;
    if (USE_OCC && !((__ldg(m.occ + (h >> 5)) >> (h & 31u)) & 1u)) return NO_BUCKET;
    Entry e = load_entry(m.table, h);
    if (e.key == KEY_EMPTY) return NO_BUCKET;
    const uint32_t reach = entry_reach(e.cr);
    for (uint32_t d = 0;; ++d) {
        if (e.key == key) {
            count = entry_count(e.cr);
            return (count && e.bucket < BUCKET_PENDING) ? e.bucket : NO_BUCKET;
        }
        if (d >= reach) break;
        e = load_entry(m.table, (h + d + 1) & m.mask);
        if (e.key == KEY_EMPTY) break;
    }
    return NO_BUCKET;
}

// lexicographic (d2, id) candidate; d2 >= 0 so its bit pattern orders like the value
struct Best {
    double d2;
    uint32_t id;
    uint32_t ref;     // bucket*cap + position of the stored point
};

__device__ __forceinline__ bool better(double d2, uint32_t id, const Best& b) {
    return d2 < b.d2 || (d2 == b.d2 && id < b.id);
}

// warp arg-min over (d2, id): redux.sync steps on the 64-bit pattern halves, and on the id only if two lanes tie on
// d2 (rare); returns the lane holding the winner (lanes with no candidate carry d2 = +inf, id = NO_ID)
__device__ __forceinline__ int warp_argmin(double d2, uint32_t id) {
    const unsigned long long bits = (unsigned long long)__double_as_longlong(d2);
    const uint32_t hi = (uint32_t)(bits >> 32), lo = (uint32_t)bits;
    const uint32_t mhi = __reduce_min_sync(FULL, hi);
    bool c = hi == mhi;
    const uint32_t mlo = __reduce_min_sync(FULL, c ? lo : 0xFFFFFFFFu);
    c = c && lo == mlo;
    unsigned b = __ballot_sync(FULL, c);
    if (b & (b - 1)) {      // more than one lane holds the minimal d2: lowest id wins (R6)
        const uint32_t mid = __reduce_min_sync(FULL, c ? id : 0xFFFFFFFFu);
        c = c && id == mid;
        b = __ballot_sync(FULL, c);
    }
    return __ffs(b) - 1;
}

__device__ __forceinline__ int warp_incl_scan(int v, int lane) {
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const int o = __shfl_up_sync(FULL, v, d);
        if (lane >= d) v += o;
    }
    return v;
}

// The 27-voxel probe of one query by one warp (Fig. 3): lane l < 27 looks up neighbour
// (l/9-1, (l/3)%3-1, l%3-1) and keeps its bucket and count in registers.  All 32 lanes must call.
template <bool USE_OCC = false>
__device__ __forceinline__ void probe27_regs(const MapView& m, const int k[3], int lane, uint32_t& cnt, uint32_t& slot) {
    cnt = 0; slot = NO_BUCKET;
    if (lane < 27) {
        const int nx = k[0] + lane / 9 - 1, ny = k[1] + (lane / 3) % 3 - 1, nz = k[2] + lane % 3 - 1;
        if (index_in_range(nx) && index_in_range(ny) && index_in_range(nz)) slot = find_voxel<USE_OCC>(m, pack_key(nx, ny, nz), cnt);
    }
}

// ---- the flattened candidate list of one query ---------------------------------------------------------------------
// The warp sweeps the points of the voxels that matter as ONE list, 32 consecutive candidates per step, so lanes never
// idle on half-empty voxels.  Per warp in shared memory: the occupied voxels in compact form (slot, first candidate
// index) and, for every 32-candidate step, a bit mask of the positions where a new voxel starts.  Candidate j of step c
// then belongs to compact voxel (#starts in earlier steps) + popc(mask_c & lanes <= mine) - 1: two LDS and a popc
// instead of a per-lane walk over the prefix array.
constexpr int CAND_STEPS = 27 * 64 / 32;    // cap <= 64
struct __align__(16) CandList {
    int off[32];                 // first candidate index of compact voxel c
    uint32_t slot[32];           // its bucket
    uint32_t mask[CAND_STEPS];   // voxel-start bits of step c
};

// all 32 lanes call; lane l < 27 passes the count (0 = skip) and slot of neighbour voxel l; returns the total
__device__ __forceinline__ int cand_build(CandList& L, uint32_t cnt, uint32_t slot, int lane) {
    const int incl = warp_incl_scan((int)cnt, lane);
    const int total = __shfl_sync(FULL, incl, 31);
    const unsigned occ = __ballot_sync(FULL, cnt > 0);
    const int steps = (total + 31) >> 5;
    for (int c = lane; c < steps; c += 32) L.mask[c] = 0u;
    __syncwarp();
    if (cnt > 0) {
        const int excl = incl - (int)cnt;
        const int ci = __popc(occ & ((1u << lane) - 1u));
        L.off[ci] = excl;
        L.slot[ci] = slot;
        atomicOr(&L.mask[excl >> 5], 1u << (excl & 31));
    }
    __syncwarp();
    return total;
}

// iteration state of one lane over the list: call cand_next once per 32-candidate step, in order
struct CandIter { int before; };   // voxel starts in earlier steps
__device__ __forceinline__ uint32_t cand_next(const CandList& L, CandIter& it, int step, int j, int lane, int cap) {
    const uint32_t mk = L.mask[step];
    const int v = it.before + __popc(mk & (0xFFFFFFFFu >> (31 - lane))) - 1;
    it.before += __popc(mk);
    return L.slot[v] * (uint32_t)cap + (uint32_t)(j - L.off[v]);
}

// warp-wide minimum of a non-negative double (its bit pattern orders like its value): two redux.sync steps
__device__ __forceinline__ double warp_min_nonneg(double d2) {
    const unsigned long long bits = (unsigned long long)__double_as_longlong(d2);
    const uint32_t hi = (uint32_t)(bits >> 32), lo = (uint32_t)bits;
    const uint32_t mhi = __reduce_min_sync(FULL, hi);
    const uint32_t mlo = __reduce_min_sync(FULL, hi == mhi ? lo : 0xFFFFFFFFu);
    return __longlong_as_double((long long)(((unsigned long long)mhi << 32) | mlo));
}

// Lower bound of the squared distance from q (inside voxel k) to ANY point stored in neighbour voxel
// k + (ox, oy, oz).  A point of voxel index K along one axis satisfies K v - e <= p < (K + 1) v + e with
// e < (|K| + 1) v 2^-24 (the key is the floor of ONE rounded fp32 quotient, R1), so the faces are pulled in by a
// margin of (|k| + 2) v 2^-20, which also covers the rounding of the bound itself.  k v is exact in binary64.
__device__ __forceinline__ double voxel_lower_bound(float qx, float qy, float qz, const int k[3], float v, int ox, int oy, int oz) {
    const double dv = (double)v;
    const double q[3] = {(double)qx, (double)qy, (double)qz};
    const int o[3] = {ox, oy, oz};
    double lb = 0.0;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const double margin = (double)(abs(k[a]) + 2) * dv * 9.5367431640625e-07;   // 2^-20
        double gap = 0.0;
        if (o[a] < 0) gap = q[a] - (double)k[a] * dv - margin;
        else if (o[a] > 0) gap = (double)(k[a] + 1) * dv - q[a] - margin;
        gap = fmax(gap, 0.0);
        lb += gap * gap;
    }
    return lb;
}

// A6 by one warp, all 32 lanes must call; every lane returns the winner (best.id == NO_ID if none) and its
// coordinates.  Exactly the 27-voxel (d2, id)-minimum of R6, reached with fewer reads: the query's own voxel is
// swept first, then a neighbour voxel is read only if its lower bound does not exceed the best d2 so far
// (a skipped voxel holds only points strictly farther than the current best, so it cannot change the result,
// ties included).  The surviving voxels are swept as ONE flattened candidate list, 32 float4 per step.
template <bool USE_OCC = false>
__device__ __forceinline__ Best warp_nearest(const MapView& m, float qx, float qy, float qz, const int k[3], int lane,
                                             CandList& L, float& rx, float& ry, float& rz) {
    uint32_t cnt, slot;
    probe27_regs<USE_OCC>(m, k, lane, cnt, slot);
    Best best;
    best.d2 = __longlong_as_double(0x7FF0000000000000ll);
    best.id = NO_ID;
    best.ref = 0;
    float bx = 0.f, by = 0.f, bz = 0.f;
    // few occupied voxels (the rule at small voxel sizes: 2 of 27 on the 20 M-point map at v = 0.25): sweep them one after
    // the other -- bounding and flattening would cost more instructions than the handful of candidates they could save
    unsigned occv = __ballot_sync(FULL, cnt > 0);
    if (__popc(occv) <= 4) {
        while (occv) {
            const int l = __ffs(occv) - 1;
            occv &= occv - 1;
            const uint32_t c = __shfl_sync(FULL, cnt, l), b = __shfl_sync(FULL, slot, l);
            for (uint32_t j = lane; j < c; j += 32) {
                const uint32_t ref = b * (uint32_t)m.cap + j;
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
    const uint32_t c_cnt = __shfl_sync(FULL, cnt, 13), c_slot = __shfl_sync(FULL, slot, 13);
    for (uint32_t j = lane; j < c_cnt; j += 32) {
        const uint32_t ref = c_slot * (uint32_t)m.cap + j;
        const float4 p = __ldg(m.points + ref);
        const double d2 = dist2(qx, qy, qz, p.x, p.y, p.z);
        const uint32_t id = __float_as_uint(p.w);
        if (better(d2, id, best)) { best.d2 = d2; best.id = id; best.ref = ref; bx = p.x; by = p.y; bz = p.z; }
    }
    const double bound = warp_min_nonneg(best.d2);
    uint32_t c2 = 0;
    if (lane < 27 && lane != 13 && cnt > 0) {
        const double lb = voxel_lower_bound(qx, qy, qz, k, m.voxel, lane / 9 - 1, (lane / 3) % 3 - 1, lane % 3 - 1);
        if (lb <= bound) c2 = cnt;
    }
    const int total = cand_build(L, c2, slot, lane);
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

}  // namespace far
