// far_map.cu -- the voxel hashmap: create / clear / deterministic capped insert / prune + in-place rehash / export / stats.
//
// PAPER.md:62-68 (cuVoxelMap: custom key = 3D voxel indices, linear probing, <= N_max points per voxel, built
// for concurrent access), PAPER.md:109 (submap update: insert at T_L with a per-voxel cap, recompute the
// covariances of added points only, remove voxels beyond a range limit), PAPER.md:171,186 (everything
// preallocated: allocations show up as latency peaks).
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
//
// Storage (far_common.cuh): 16-byte table entries {key, bucket, count | reach}, buckets in a DENSE pool handed out by a
// bump allocator + free list.  Pruning returns buckets at once and leaves dead keys behind; when their number passes a
// device-side threshold the prune call's follow-up kernel rebuilds the entries into the shadow table and copies them
// back.  Nothing on this path allocates, frees or synchronises.
#include <algorithm>
#include <atomic>
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

__device__ __forceinline__ uint32_t ld_volatile(const uint32_t* p) { return *reinterpret_cast<const volatile uint32_t*>(p); }

__device__ __forceinline__ Entry ld_entry_volatile(const Entry* p) {
    uint4 raw;
    asm volatile("ld.volatile.global.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(raw.x), "=r"(raw.y), "=r"(raw.z), "=r"(raw.w) : "l"(p) : "memory");
    Entry e;
    e.key = ((unsigned long long)raw.y << 32) | raw.x;
    e.bucket = raw.z;
    e.cr = raw.w;
    return e;
}

// raise the reach of home slot h to at least r, leaving the count byte alone (only for DISPLACED keys: a key sitting in
// its home slot needs no reach)
__device__ __forceinline__ void raise_reach(Entry* table, uint32_t h, uint32_t r) {
    uint32_t* w = &table[h].cr;
    uint32_t old = ld_volatile(w);
    while (entry_reach(old) < r) {
        const uint32_t seen = atomicCAS(w, old, (r << 8) | (old & 0xFFu));
        if (seen == old) break;
        old = seen;
    }
}

// find `key` or claim an empty slot for it: 64-bit atomicCAS on the key word, linear probing step 1.
// One 16-byte load per probed slot yields key, bucket and count together (the two 8-byte halves may be of different age:
// harmless, a stale half only sends the caller through the slower path).  Returns NO_SLOT if the key is absent and the
// table takes no more keys; `e` = the entry as seen (bucket = BUCKET_PENDING on a slot claimed just now).
__device__ __forceinline__ uint32_t find_or_claim(Entry* table, uint32_t mask, uint32_t slots, unsigned long long key,
                                                  bool may_claim, bool& claimed, Entry& e, uint32_t first_probe = 0,
                                                  uint32_t* occ = nullptr) {
    // first_probe: slots h .. h + first_probe - 1 are known to hold other keys (keys never leave a slot while inserts run)
    const uint32_t h = hash_key(key) & mask;
    uint32_t s = (h + first_probe) & mask;
    claimed = false;
    for (uint32_t probes = first_probe; probes < slots; ++probes) {
        e = ld_entry_volatile(table + s);
        if (e.key == KEY_EMPTY) {
            if (!may_claim || probes >= 0xFFFFFEu) return NO_SLOT;
            const unsigned long long cur = atomicCAS(&table[s].key, KEY_EMPTY, key);
            if (cur == KEY_EMPTY) {
                claimed = true;
                if (occ) atomicOr(&occ[s >> 5], 1u << (s & 31u));   // the slot holds a key from now on (far_common.cuh)
                e.key = key; e.bucket = BUCKET_PENDING; e.cr &= ~0xFFu;
                if (probes) raise_reach(table, h, probes);   // keep the reach of the key's home slot up to date (find_voxel)
                return s;
            }
            if (cur == key) { e = ld_entry_volatile(table + s); return s; }
        } else if (e.key == key) {
            return s;
        }
        s = (s + 1) & mask;
    }
    return NO_SLOT;
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

// ---- regular spacing ("regularly spaced ... minimum point-to-point distance of ~65 cm"; R21) --
// With min_spacing > 0 acceptance depends on the points accepted before, so the atomicMin chain cannot decide it.  The
// claim kernel then only LISTS every offered point for its voxel (count per bucket, bucket per point); the offers of a
// voxel are gathered into one contiguous segment (scan + scatter) and one block per touched voxel sorts them by id and
// walks them in order, 32 at a time against the stored points (spaced_commit_kernel).  Scratch allocated at create.
struct Spaced {
    uint32_t* offer_cnt;       // [max_voxels] offers per bucket in the running chunk (all zero between chunks)
    uint32_t* voxel_t;         // [max_voxels] index of the bucket's voxel in the touched list
    uint32_t* pt_bucket;       // [max_batch]  bucket of point i of the chunk, NO_BUCKET if it is not offered
    uint32_t* seg_start;       // [max_batch + 1] first entry of touched voxel t in `seg`
    uint32_t* seg;             // [max_batch]  point indices, grouped by voxel
    double s2;                 // min_spacing^2
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

// ---- insert, kernel 1: key -> find-or-claim -> bucket -> atomicMin chain --------------------------------------------
// All 32 lanes of a warp stay in the kernel to its end (no early return), so every collective below uses the full mask.
// Lanes that offer points to the SAME voxel (a LiDAR ring crossing a voxel gives a run of consecutive ids; 73 % of a C2
// scan falls into voxels that are offered more than cap points, up to 700) elect one leader: only the leader walks the
// table, and the lanes' ranks `ahead` let each id enter the chain at c0 + ahead instead of at c0 (exact: an id may enter
// anywhere at or before its final position -- every position still ends up with the minimum of the ids that reach it --
// and it removes most of the shifting); if c0 + ahead is already past the limit the point cannot survive at all.
__global__ void __launch_bounds__(256) insert_claim_chain_kernel(MapView m, const float* __restrict__ xyz, int64_t n,
                                                                  const int64_t* __restrict__ d_n, int stride, int pose_mode, Pose hpose,
                                                                  const Pose* __restrict__ d_pose, uint32_t id_offset,
                                                                  uint32_t* __restrict__ touched, Asmd asmd, Spaced sp) {
    // Every counter of the map sits in one 128-byte line of L2, and the L2 retires about one atomic per 1.3 cycles on a line:
    // one atomic per WARP and counter (3,656 warps for a 117k-point scan, six counters) held the whole kernel back by ~14 us.
    // So everything is summed per BLOCK in shared memory first: the block draws its buckets with ONE atomic after a barrier
    // that only waits for the lookups, and its statistics go out with one atomic each from whichever warp finishes last.
    __shared__ uint32_t s_cnt[10];              // 0 buckets wanted, 1 new keys, 2 invalid, 3 opened, 4 dropped, 5 warps done, 6 draw base,
                                                // 7 dead keys revived, 8 new keys left without a bucket
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
    const unsigned lt = (1u << lane) - 1u;
    const Pose& T = (pose_mode == 2) ? *d_pose : hpose;
    Counters* ctr = m.ctr;
    if (threadIdx.x < 10) s_cnt[threadIdx.x] = 0u;
    __syncthreads();
    if (d_n) n = min(n, *d_n);                  // frame graph: launch sized for the largest scan, count on the device
    float p[3];
    int k[3] = {0, 0, 0};
    bool valid = false, bad = false;
    if (i < n) {
        valid = load_pose_point(xyz, i, stride, pose_mode, T, p) && voxel_index(p[0], p[1], p[2], m.voxel, k);
        bad = !valid;
    }
    // invalid lanes get distinct fake keys (bit 63 is never set by a valid key)
    const unsigned long long key = valid ? pack_key(k[0], k[1], k[2]) : ((1ull << 63) | (unsigned long long)lane);
    const unsigned same = __match_any_sync(FULL, key);
    const uint32_t ahead = __popc(same & lt);

    // phase 1: every lane looks its voxel up by itself, read-only; the probe's 16-byte load brings bucket and count along.
    // On a map that already holds the scan's voxels (the submap update of a frame) every lane is done here and goes
    // straight to its chain -- nobody waits for a neighbour's slower walk.
    uint32_t s = NO_SLOT, b = NO_BUCKET, c0 = 0;
    bool claimed = false, want = false, resolved = !valid;
    const uint32_t id_base = (uint32_t)ctr->next_id + id_offset;           // requested early: needed by the chain only
    uint32_t walked = 0;                        // slots of the read-only walk that held OTHER keys: the claim resumes behind them
    // the allocator's state does not change while the kernel runs: fetched now, with the id counter (same line), not when
    // a bucket is drawn
    const uint32_t nf = (uint32_t)ctr->n_free, bump0 = ctr->bump;
    if (valid) {
        uint32_t t = hash_key(key) & m.mask;
        for (uint32_t probes = 0; probes < m.slots; ++probes) {
            const Entry e = ld_entry_volatile(m.table + t);
            if (e.key == key) {
                if (e.bucket < BUCKET_PENDING) { s = t; b = e.bucket; c0 = entry_count(e.cr); resolved = true; }
                break;
            }
            if (e.key == KEY_EMPTY) break;
            t = (t + 1) & m.mask;
            walked = probes + 1;
        }
    }
    // phase 1b (only warps with an unresolved lane): the voxel is new, dead or being opened by someone else.  One leader
    // per voxel claims the key / the right to allocate; the others of its group get the result by shuffle.
    const unsigned unresolved = __ballot_sync(FULL, !resolved);
    const bool is_leader = !resolved && (__ffs(same & unresolved) - 1) == lane;
    if (unresolved && is_leader) {
        const bool may_claim = ctr->n_keys < m.key_limit;                  // enforced up to the keys claimed while this runs
        Entry e;
        s = find_or_claim(m.table, m.mask, m.slots, key, may_claim, claimed, e, walked, m.occ);
        if (s != NO_SLOT) {
            b = e.bucket;
            c0 = entry_count(e.cr);                                        // stable: only the commit kernel writes counts
            // a voxel without a bucket gets one from exactly one thread of the grid: the claimer of a new key (its bucket
            // word starts out PENDING), or whoever wins the NO_BUCKET -> PENDING exchange on the dead key of a pruned voxel
            want = claimed;
            if (b == NO_BUCKET) {
                const uint32_t old = atomicCAS(&m.table[s].bucket, NO_BUCKET, BUCKET_PENDING);
                if (old == NO_BUCKET) want = true; else b = old;
            }
        }
    }
    // phase 2: the BLOCK's allocators draw together: ONE atomic; the first n_free draws of a kernel come off the free list,
    // the rest from the fresh end of the pool (n_free and bump do not change while the kernel runs)
    const unsigned newk = __ballot_sync(FULL, claimed);
    const unsigned wm = __ballot_sync(FULL, want);
    uint32_t woff = 0;
    if (lane == 0) {
        if (newk) atomicAdd(&s_cnt[1], (uint32_t)__popc(newk));
        if (wm) woff = atomicAdd(&s_cnt[0], (uint32_t)__popc(wm));
    }
    woff = __shfl_sync(FULL, woff, 0);
    __syncthreads();                            // (nobody waits for anybody before this point: the lookups and claims only)
    if (threadIdx.x == 0) {
        if (s_cnt[0]) s_cnt[6] = atomicAdd(&ctr->n_alloc, s_cnt[0]);
        if (s_cnt[1]) atomicAdd(&ctr->n_keys, s_cnt[1]);
    }
    __syncthreads();
    bool opened = false;
    if (wm) {
        if (want) {
            const uint32_t a = s_cnt[6] + woff + __popc(wm & lt);
            if (a < nf) b = m.free_list[nf - 1u - a];
            else {
                b = bump0 + (a - nf);
                if (b >= m.max_buckets) b = NO_BUCKET;                  // pool exhausted: the voxel stays without points
            }
            atomicExch(&m.table[s].bucket, b);
            opened = b != NO_BUCKET;
            c0 = 0;
        }
    }
    // phase 3: another thread may be allocating this voxel's bucket right now; it never waits for anything, so this ends
    bool fresh_voxel = false;
    if (unresolved) {
        if (is_leader && s != NO_SLOT && !want) {
            while (b == BUCKET_PENDING) b = ld_volatile(&m.table[s].bucket);
        }
        const unsigned grp = same & unresolved;                 // the lanes that wait for this voxel's leader (or nobody)
        const int leader = __ffs(grp) - 1;
        if (!resolved) {
            s = __shfl_sync(grp, s, leader);
            b = __shfl_sync(grp, b, leader);
            c0 = __shfl_sync(grp, c0, leader);
            fresh_voxel = __shfl_sync(grp, (int)want, leader) != 0;
        }
    }

    // statistics: per block in shared memory; flushed at the end of the kernel by the warp that finishes last
    const unsigned m_bad = __ballot_sync(FULL, bad);
    const unsigned m_drop = __ballot_sync(FULL, valid && b == NO_BUCKET);
    const unsigned m_open = __ballot_sync(FULL, opened);
    // Counters::n_dead = keys in the table that own no bucket: the dead key of a pruned voxel that got a bucket again leaves
    // that set, a new key the exhausted pool had no bucket for is born into it
    const unsigned m_rev = __ballot_sync(FULL, want && !claimed && opened);
    const unsigned m_still = __ballot_sync(FULL, want && claimed && !opened);
    if (lane == 0) {
        if (m_bad) atomicAdd(&s_cnt[2], (uint32_t)__popc(m_bad));
        if (m_open) atomicAdd(&s_cnt[3], (uint32_t)__popc(m_open));
        if (m_drop) atomicAdd(&s_cnt[4], (uint32_t)__popc(m_drop));
        if (m_rev) atomicAdd(&s_cnt[7], (uint32_t)__popc(m_rev));
        if (m_still) atomicAdd(&s_cnt[8], (uint32_t)__popc(m_still));
    }

    // phase 4: the chain.  cap = this voxel's limit: the fixed cap, or N_ASMD (positions at and beyond it are never written)
    bool first_of_voxel = false;
    if (sp.on) {
        // regular spacing: no chain -- the point is listed for its voxel (one atomic per group of lanes with the same key)
        uint32_t pb = NO_BUCKET;
        if (valid && b != NO_BUCKET) {
            pb = b;
            if (ahead == 0) first_of_voxel = atomicAdd(&sp.offer_cnt[b], (unsigned)__popc(same)) == 0u;
        }
        if (i < n) sp.pt_bucket[i] = pb;
    } else if (valid && b != NO_BUCKET) {
        const uint32_t cap = voxel_limit(m, asmd, k, pose_mode, T);
        uint32_t* idw = m.ids + (size_t)b * (uint32_t)m.cap;   // id word of position 0
        uint32_t x = id_base + (uint32_t)i;
        // ids at a position only ever decrease: if the last position already holds a smaller id, x cannot survive
        // (not worth a load on a voxel that was opened just now)
        if (c0 + ahead < cap && (fresh_voxel || !(ld_volatile(idw + (cap - 1)) < x))) {
            // The id words of a bucket are sorted at every instant and only ever decrease, so a position seen holding an
            // id < x will never take x: gallop over such positions with plain reads (4 independent loads per step)
            // instead of walking them with dependent atomics.  A stale read only makes the chain start earlier.
            uint32_t pos = c0 + ahead;
            while (pos + 4 <= cap) {
                if (ld_volatile(idw + (pos + 3)) < x) pos += 4; else break;
            }
            for (; pos < cap; ++pos) {
                const uint32_t old = atomicMin(idw + pos, x);
                if (old == NO_ID) {
                    first_of_voxel = pos == c0;                // unique per voxel and chunk
                    break;
                }
                if (old > x) x = old;
            }
        }
    }
    // the touched list: TOUCHED_SUBS sub-lists with their counters on separate lines (a block appends to sub-list
    // blockIdx mod TOUCHED_SUBS), so that this per-warp atomic meets ~1/32 of the grid on its line; the regular-spacing path
    // wants one flat list (its scan kernel walks it) and keeps to sub-list 0
    const unsigned m_first = __ballot_sync(FULL, first_of_voxel);
    if (m_first) {
        const uint32_t sub = sp.on ? 0u : (blockIdx.x % TOUCHED_SUBS);
        uint32_t at = 0;
        if (lane == 0) at = atomicAdd(&m.touched_cnt[sub * 32u], (unsigned)__popc(m_first));
        at = __shfl_sync(FULL, at, 0);
        if (first_of_voxel) {
            const uint32_t t = at + __popc(m_first & lt);
            touched[(size_t)sub * m.touched_sub_cap + t] = s;
            if (sp.on) sp.voxel_t[b] = t;
        }
    }
    // the block's statistics: whichever warp finishes last sends them (no barrier: nobody waits for the slowest chain)
    __syncwarp();
    bool last_warp = false;
    if (lane == 0) {
        __threadfence_block();
        last_warp = atomicAdd(&s_cnt[5], 1u) == (blockDim.x >> 5) - 1u;
    }
    if (__shfl_sync(FULL, (int)last_warp, 0) && lane == 0) {
        __threadfence_block();
        const uint32_t nb = *(volatile uint32_t*)&s_cnt[2], no = *(volatile uint32_t*)&s_cnt[3], nd = *(volatile uint32_t*)&s_cnt[4];
        if (nb) atomicAdd(&ctr->st_invalid, (unsigned long long)nb);
        if (no) atomicAdd(&ctr->st_new_voxels, (unsigned long long)no);
        if (nd) { atomicAdd(&ctr->st_dropped_full, (unsigned long long)nd); ctr->full_flag = 1u; }
        const uint32_t nr = *(volatile uint32_t*)&s_cnt[7], ns = *(volatile uint32_t*)&s_cnt[8];
        if (nr) atomicSub(&ctr->n_dead, nr);
        if (ns) atomicAdd(&ctr->n_dead, ns);
    }
}

// The block that finishes last closes the chunk (all threads of all blocks call): touched list and allocator re-armed; after
// the last chunk the call's statistics go out, the counters are zeroed and the id counter advances -- no separate launch,
// no memset.
__device__ __forceinline__ void insert_epilogue(const MapView& m, int64_t n_call, int last_chunk, far_insert_stats_t* __restrict__ d_stats) {
    Counters* ctr = m.ctr;
    if (last_block_done(&ctr->ticket[0]) && threadIdx.x == 0) {
        volatile Counters* c = ctr;
        for (uint32_t j = 0; j < TOUCHED_SUBS; ++j) m.touched_cnt[j * 32u] = 0u;
        if (last_chunk) { c->n_tasks = c->n_cov; c->n_cov = 0u; }
        {   // fold the kernel's bucket draws into the allocator state
            const unsigned drawn = c->n_alloc, nf = (unsigned)c->n_free;
            const unsigned from_free = drawn < nf ? drawn : nf;
            c->n_free = (int)(nf - from_free);
            const unsigned long long bump = (unsigned long long)c->bump + (drawn - from_free);
            c->bump = bump > m.max_buckets ? m.max_buckets : (unsigned)bump;
            c->n_alloc = 0u;
        }
        if (last_chunk) {
            c->call_first_id = c->next_id;
            c->next_id = c->next_id + (unsigned long long)n_call;
            if (d_stats) {
                d_stats->n_offered = n_call;
                d_stats->n_accepted = (int64_t)c->st_accepted;
                d_stats->n_new_voxels = (int64_t)c->st_new_voxels;
                d_stats->n_dropped_full = (int64_t)c->st_dropped_full;
                d_stats->n_invalid = (int64_t)c->st_invalid;
            }
            c->st_accepted = 0ull; c->st_new_voxels = 0ull; c->st_dropped_full = 0ull; c->st_invalid = 0ull;
            if (c->full_flag) m.mail->full = 1u;
        }
    }
}

// ---- insert, kernel 2: 8 lanes per touched voxel write the coordinates of the surviving ids -------------------
// Every step of a voxel's commit is a dependent, usually cold access (touched list -> entry -> id row -> source point ->
// bucket), and most touched voxels receive a handful of points, so a warp works on FOUR voxels at once.  The block that
// finishes last closes the call: statistics out, counters re-armed, id counter advanced -- no separate launch, no memset.
constexpr int COMMIT_LANES = 8;      // 4 and 16 measure the same within 3 %
__global__ void __launch_bounds__(256) insert_commit_kernel(MapView m, const float* __restrict__ xyz, int stride,
                                                             int pose_mode, Pose hpose, const Pose* __restrict__ d_pose,
                                                             uint32_t id_offset, const uint32_t* __restrict__ touched,
                                                             uint32_t* __restrict__ cov_list, int64_t n_call, const int64_t* __restrict__ d_n,
                                                             int last_chunk, far_insert_stats_t* __restrict__ d_stats) {
    const int lane = threadIdx.x & 31, sub = lane / COMMIT_LANES, sl = lane % COMMIT_LANES;
    constexpr int PER_WARP = 32 / COMMIT_LANES;
    const unsigned gmask = ((1u << COMMIT_LANES) - 1u) << (sub * COMMIT_LANES);
    const int64_t warp = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int64_t nwarps = ((int64_t)gridDim.x * blockDim.x) >> 5;
    const Pose& T = (pose_mode == 2) ? *d_pose : hpose;
    Counters* ctr = m.ctr;
    // warp w serves sub-list w mod TOUCHED_SUBS (the claim kernel dealt its blocks over the sub-lists: they are balanced)
    const uint32_t sub_list = (uint32_t)(warp % TOUCHED_SUBS);
    const int64_t per_list = nwarps / TOUCHED_SUBS;      // warps per sub-list (warps beyond per_list * TOUCHED_SUBS idle)
    const uint32_t n_touched = warp < per_list * TOUCHED_SUBS ? m.touched_cnt[sub_list * 32u] : 0u;
    touched += (size_t)sub_list * m.touched_sub_cap;
    const uint32_t first_id = (uint32_t)ctr->next_id + id_offset;
    const uint32_t cap = (uint32_t)m.cap;
    if (d_n) n_call = min(n_call, *d_n);
    unsigned long long acc_new = 0;                       // lane sl == 0 of each group: points accepted
    for (int64_t t0 = (warp / TOUCHED_SUBS) * PER_WARP; t0 < n_touched; t0 += per_list * PER_WARP) {
        const int64_t t = t0 + sub;
        const bool active = t < n_touched;
        uint32_t s = 0, b = 0, cr = 0, c0 = cap;
        unsigned long long vkey = 0;
        if (active) {
            s = touched[t];
            const Entry e = m.table[s];
            b = e.bucket; cr = e.cr; vkey = e.key;
            c0 = entry_count(cr);
        }
        uint32_t n_new = 0;
        for (uint32_t step = 0; step * COMMIT_LANES < cap; ++step) {      // warp-uniform trip count
            const uint32_t pos = c0 + step * COMMIT_LANES + sl;
            uint32_t id = NO_ID;
            if (active && pos < cap) id = m.ids[(size_t)b * cap + pos];
            const bool is_new = id != NO_ID;
            if (is_new) {
                float p[3];
                load_pose_point(xyz, (int64_t)(id - first_id), stride, pose_mode, T, p);
                m.points[(size_t)b * cap + pos] = make_float4(p[0], p[1], p[2], __uint_as_float(id));
                if (m.cov_ok) m.cov_ok[(size_t)b * cap + pos] = 0;
            }
            const unsigned bal = __ballot_sync(FULL, is_new);
            if (bal == 0) break;                                           // ids fill positions in order: nothing further
            n_new += __popc(bal & gmask);
        }
        if (active && sl == 0) {
            m.table[s].cr = (cr & ~0xFFu) | (c0 + n_new);
            acc_new += n_new;
        }
        if (cov_list != nullptr) {
            // one covariance task per voxel that received points: {key, bucket, c0 | n_new << 8} (far_query.cu serves a voxel's
            // new points together: they share their 27-voxel candidate set)
            const bool has = active && sl == 0 && n_new > 0;
            const unsigned tb = __ballot_sync(FULL, has);
            if (tb) {
                uint32_t at = 0;
                if (lane == 0) at = atomicAdd(&ctr->n_cov, (uint32_t)__popc(tb));
                at = __shfl_sync(FULL, at, 0);
                if (has) reinterpret_cast<uint4*>(cov_list)[at + __popc(tb & ((1u << lane) - 1u))] = make_uint4((uint32_t)vkey, (uint32_t)(vkey >> 32), b, c0 | (n_new << 8));
            }
        }
    }
    // accepted points: per block in shared memory, one atomic on the map's counter line per block
    __shared__ unsigned long long s_accepted;
    if (threadIdx.x == 0) s_accepted = 0ull;
    __syncthreads();
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) acc_new += __shfl_xor_sync(FULL, acc_new, d);
    if (lane == 0 && acc_new) atomicAdd(&s_accepted, acc_new);
    __syncthreads();
    if (threadIdx.x == 0 && s_accepted) atomicAdd(&ctr->st_accepted, s_accepted);

    insert_epilogue(m, n_call, last_chunk, d_stats);
}

// ---- regular spacing, kernel 2: exclusive scan of the offers per touched voxel (one block; a few thousand voxels) -----
__global__ void __launch_bounds__(1024) spaced_scan_kernel(MapView m, const uint32_t* __restrict__ touched, Spaced sp) {
    __shared__ uint32_t s_warp[32];
    __shared__ uint32_t s_carry;
    if (threadIdx.x == 0) s_carry = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const uint32_t n_touched = m.touched_cnt[0];              // regular spacing: the flat list = sub-list 0
    for (uint32_t base = 0; base < n_touched; base += 1024) {
        const uint32_t t = base + threadIdx.x;
        const uint32_t c = t < n_touched ? sp.offer_cnt[m.table[touched[t]].bucket] : 0u;
        uint32_t incl = c;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const uint32_t o = __shfl_up_sync(FULL, incl, d);
            if (lane >= d) incl += o;
        }
        if (lane == 31) s_warp[wid] = incl;
        __syncthreads();
        if (wid == 0) {
            uint32_t x = s_warp[lane];
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const uint32_t o = __shfl_up_sync(FULL, x, d);
                if (lane >= d) x += o;
            }
            s_warp[lane] = x;
        }
        __syncthreads();
        const uint32_t excl = s_carry + (wid ? s_warp[wid - 1] : 0u) + incl - c;
        if (t < n_touched) sp.seg_start[t] = excl;
        __syncthreads();
        if (threadIdx.x == 1023) s_carry = excl + c;
        __syncthreads();
    }
    if (threadIdx.x == 0) sp.seg_start[n_touched] = s_carry;
}

// ---- regular spacing, kernel 3: every offered point goes into its voxel's segment (order inside a segment arbitrary) --
__global__ void __launch_bounds__(256) spaced_scatter_kernel(MapView m, int64_t n, const int64_t* __restrict__ d_n, Spaced sp) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (d_n) n = min(n, *d_n);
    if (i >= n) return;
    const uint32_t b = sp.pt_bucket[i];
    if (b == NO_BUCKET) return;
    const uint32_t pos = atomicSub(&sp.offer_cnt[b], 1u) - 1u;          // counts down to zero: clean for the next chunk
    sp.seg[sp.seg_start[sp.voxel_t[b]] + pos] = (uint32_t)i;
}

// ---- regular spacing, kernel 4: one block per touched voxel sorts its offers by id and walks them in order -----------
// The walk is the sequential rule of R21 (accept iff the voxel holds fewer points than its limit and none of them is
// closer than min_spacing, FP64 d2 of R6, strict <), 32 offers at a time: every lane tests its offer against the stored
// points; the lowest passing lane is accepted, the lanes after it re-test against that one point, and so on.  Segments
// longer than the sort buffer are cut into id ranges (halved until they fit).
constexpr int SP_THREADS = 128;
constexpr int SP_SORT = 4096;        // offers sorted at a time
__global__ void __launch_bounds__(SP_THREADS) spaced_commit_kernel(MapView m, const float* __restrict__ xyz, int64_t n_chunk, int stride,
                                                                   int pose_mode, Pose hpose, const Pose* __restrict__ d_pose,
                                                                   uint32_t id_offset, const uint32_t* __restrict__ touched,
                                                                   uint32_t* __restrict__ cov_list, int64_t n_call,
                                                                   const int64_t* __restrict__ d_n, int last_chunk,
                                                                   far_insert_stats_t* __restrict__ d_stats, Asmd asmd, Spaced sp) {
    __shared__ uint32_t s_buf[SP_SORT];
    __shared__ float4 s_pts[64];
    __shared__ uint32_t s_count, s_n, s_nacc;
    const Pose& T = (pose_mode == 2) ? *d_pose : hpose;
    Counters* ctr = m.ctr;
    if (d_n) { n_call = min(n_call, *d_n); n_chunk = min(n_chunk, *d_n); }
    const uint32_t first_id = (uint32_t)ctr->next_id + id_offset;
    const uint32_t n_touched = m.touched_cnt[0];
    const uint32_t cap = (uint32_t)m.cap;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    for (uint32_t t = blockIdx.x; t < n_touched; t += gridDim.x) {
        const uint32_t s = touched[t];
        const Entry e = m.table[s];
        const uint32_t b = e.bucket, c0 = entry_count(e.cr);
        int k[3];
        unpack_key(e.key, k);
        const uint32_t limit = voxel_limit(m, asmd, k, pose_mode, T);
        const uint32_t seg0 = sp.seg_start[t], L = sp.seg_start[t + 1] - seg0;
        __syncthreads();
        if (threadIdx.x < c0) s_pts[threadIdx.x] = m.points[(size_t)b * cap + threadIdx.x];
        if (threadIdx.x == 0) { s_count = c0; s_nacc = 0; }
        __syncthreads();
        // id ranges [lo, hi) of point indices, each holding at most SP_SORT of the voxel's offers
        uint32_t lo = 0;
        while (lo < (uint32_t)n_chunk && s_count < limit) {
            uint32_t hi = (uint32_t)n_chunk;
            for (;;) {
                if (threadIdx.x == 0) s_n = 0;
                __syncthreads();
                uint32_t mine = 0;
                for (uint32_t j = threadIdx.x; j < L; j += SP_THREADS) { const uint32_t v = sp.seg[seg0 + j]; mine += (v >= lo && v < hi); }
                mine = __reduce_add_sync(FULL, mine);
                if (lane == 0 && mine) atomicAdd(&s_n, mine);
                __syncthreads();
                const uint32_t cnt = s_n;
                __syncthreads();
                if (cnt <= SP_SORT) break;
                hi = lo + (hi - lo) / 2;                      // cnt > SP_SORT >= 1 distinct indices: the range can be halved
            }
            // gather the range, pad to a power of two, bitonic sort ascending
            if (threadIdx.x == 0) s_n = 0;
            __syncthreads();
            for (uint32_t j = threadIdx.x; j < L; j += SP_THREADS) {
                const uint32_t v = sp.seg[seg0 + j];
                if (v >= lo && v < hi) s_buf[atomicAdd(&s_n, 1u)] = v;
            }
            __syncthreads();
            const uint32_t cnt = s_n;
            uint32_t np2 = 32;
            while (np2 < cnt) np2 <<= 1;
            for (uint32_t j = cnt + threadIdx.x; j < np2; j += SP_THREADS) s_buf[j] = NO_ID;
            __syncthreads();
            for (uint32_t kk = 2; kk <= np2; kk <<= 1) {
                for (uint32_t jj = kk >> 1; jj > 0; jj >>= 1) {
                    for (uint32_t idx = threadIdx.x; idx < np2; idx += SP_THREADS) {
                        const uint32_t ixj = idx ^ jj;
                        if (ixj > idx) {
                            const uint32_t a = s_buf[idx], c = s_buf[ixj];
                            const bool up = (idx & kk) == 0;
                            if ((a > c) == up) { s_buf[idx] = c; s_buf[ixj] = a; }
                        }
                    }
                    __syncthreads();
                }
            }
            // the walk, by warp 0
            if (wid == 0) {
                uint32_t count = s_count, nacc = s_nacc;
                for (uint32_t base = 0; base < cnt && count < limit; base += 32) {
                    const uint32_t i = base + lane < cnt ? s_buf[base + lane] : NO_ID;
                    float p[3] = {0.f, 0.f, 0.f};
                    bool pass = false;
                    if (i != NO_ID) {
                        load_pose_point(xyz, (int64_t)i, stride, pose_mode, T, p);     // valid: it has a key
                        pass = true;
                        for (uint32_t j = 0; j < count; ++j) {
                            const float4 q = s_pts[j];
                            if (dist2(p[0], p[1], p[2], q.x, q.y, q.z) < sp.s2) { pass = false; break; }
                        }
                    }
                    unsigned pm = __ballot_sync(FULL, pass);
                    while (pm && count < limit) {
                        const int w = __ffs(pm) - 1;                                   // lowest id that still passes: accepted
                        const float ax = __shfl_sync(FULL, p[0], w), ay = __shfl_sync(FULL, p[1], w), az = __shfl_sync(FULL, p[2], w);
                        if (lane == w) {
                            const uint32_t id = first_id + i;
                            const float4 np = make_float4(p[0], p[1], p[2], __uint_as_float(id));
                            s_pts[count] = np;
                            m.points[(size_t)b * cap + count] = np;
                            m.ids[(size_t)b * cap + count] = id;
                            if (m.cov_ok) m.cov_ok[(size_t)b * cap + count] = 0;
                            pass = false;
                        }
                        ++count; ++nacc;
                        if (pass && lane > w && dist2(p[0], p[1], p[2], ax, ay, az) < sp.s2) pass = false;
                        __syncwarp();
                        pm = __ballot_sync(FULL, pass) & ~((2u << w) - 1u);            // lanes after w that still pass
                    }
                }
                if (lane == 0) { s_count = count; s_nacc = nacc; }
            }
            __syncthreads();
            lo = hi;
        }
        // the voxel's new count, its accepted points into the covariance queue, the statistics
        const uint32_t nacc = s_nacc;
        if (threadIdx.x == 0) {
            m.table[s].cr = (e.cr & ~0xFFu) | s_count;
            if (nacc) atomicAdd(&ctr->st_accepted, (unsigned long long)nacc);
            // accepted points take consecutive positions c0 .. c0 + nacc - 1: one covariance task for the voxel
            if (cov_list != nullptr && nacc) reinterpret_cast<uint4*>(cov_list)[atomicAdd(&ctr->n_cov, 1u)] = make_uint4((uint32_t)e.key, (uint32_t)(e.key >> 32), b, c0 | (nacc << 8));
        }
        __syncthreads();
    }
    insert_epilogue(m, n_call, last_chunk, d_stats);
}

// ---- A5 prune (R5): thread per slot, FP64 squared centre distance, strict > -------------------
// A removed voxel's bucket goes back to the free list at once (block-aggregated push) and its key stays as a dead key.
// The last block writes the statistics and decides, from the number of dead keys, whether the rehash kernel that
// follows this one in the stream does its work or returns immediately.
__global__ void __launch_bounds__(256) prune_kernel(MapView m, double cx, double cy, double cz, const Pose* d_pose,
                                                     double r2, far_prune_stats_t* __restrict__ out) {
    __shared__ uint32_t s_wbase[8];
    __shared__ uint32_t s_base;
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    unsigned long long vr = 0, pr = 0, vl = 0, pl = 0;
    if (d_pose) { cx = d_pose->t[0]; cy = d_pose->t[1]; cz = d_pose->t[2]; }
    const double v = (double)m.voxel;
    // grid-stride over the table with one resident wave: the fence + ticket of the epilogue is paid once per block, and a
    // block's statistics are summed in registers before they touch shared memory.  A thread takes PRUNE_U slots per pass,
    // their entries requested together (a 16-byte load per thread and pass left the kernel waiting on one DRAM round trip
    // after the other: 0.6 TB/s on a frame-sized table)
    constexpr int PRUNE_U = 4;
    for (uint32_t s0 = blockIdx.x * blockDim.x * PRUNE_U; s0 < m.slots; s0 += gridDim.x * blockDim.x * PRUNE_U) {
        Entry ent[PRUNE_U];
#pragma unroll
        for (int u = 0; u < PRUNE_U; ++u) {
            const uint32_t s = s0 + u * blockDim.x + threadIdx.x;
            ent[u].key = KEY_EMPTY; ent[u].bucket = NO_BUCKET; ent[u].cr = 0;
            if (s < m.slots) ent[u] = m.table[s];
        }
        uint32_t freed[PRUNE_U];
        bool any_freed = false;
#pragma unroll
        for (int u = 0; u < PRUNE_U; ++u) {
            const uint32_t s = s0 + u * blockDim.x + threadIdx.x;
            const Entry e = ent[u];
            freed[u] = NO_BUCKET;
            const uint32_t cnt = entry_count(e.cr);
            if (e.key != KEY_EMPTY && e.bucket < BUCKET_PENDING && cnt > 0) {
                int k[3];
                unpack_key(e.key, k);
                const double dx = __dadd_rn(__dmul_rn(__dadd_rn((double)k[0], 0.5), v), -cx);
                const double dy = __dadd_rn(__dmul_rn(__dadd_rn((double)k[1], 0.5), v), -cy);
                const double dz = __dadd_rn(__dmul_rn(__dadd_rn((double)k[2], 0.5), v), -cz);
                const double d2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
                if (d2 > r2) {
                    // the id words go back to +inf so that the bucket's next owner starts clean
                    for (uint32_t j = 0; j < cnt; ++j) {
                        m.ids[(size_t)e.bucket * m.cap + j] = NO_ID;
                        if (m.cov_ok) m.cov_ok[(size_t)e.bucket * m.cap + j] = 0;
                    }
                    m.table[s].bucket = NO_BUCKET;
                    m.table[s].cr = e.cr & ~0xFFu;
                    freed[u] = e.bucket;
                    any_freed = true;
                    vr += 1; pr += cnt;
                } else {
                    vl += 1; pl += cnt;
                }
            }
        }
        // free-list push, aggregated over the block: ONE atomic on the map's counter line per block and pass (a bulk prune
        // frees a bucket in almost every lane: one atomic per warp there is a million atomics on one line of L2); a pass
        // that frees nothing -- nearly every pass of a frame's prune -- costs one barrier
        if (__syncthreads_or(any_freed)) {
            uint32_t mine = 0;
#pragma unroll
            for (int u = 0; u < PRUNE_U; ++u) mine += freed[u] != NO_BUCKET;
            const uint32_t incl = (uint32_t)warp_incl_scan((int)mine, lane);
            if (lane == 31) s_wbase[wib] = incl;
            __syncthreads();
            if (threadIdx.x == 0) {
                uint32_t tot = 0;
#pragma unroll
                for (int w = 0; w < 8; ++w) { const uint32_t c = s_wbase[w]; s_wbase[w] = tot; tot += c; }
                s_base = tot ? (uint32_t)atomicAdd(&m.ctr->n_free, (int)tot) : 0u;
            }
            __syncthreads();
            uint32_t at = s_base + s_wbase[wib] + incl - mine;
#pragma unroll
            for (int u = 0; u < PRUNE_U; ++u) if (freed[u] != NO_BUCKET) m.free_list[at++] = freed[u];
            __syncthreads();                                // s_wbase is rewritten by the next pass
        }
    }
    // block-aggregate the four statistics: one atomic per block each
    __shared__ unsigned long long s_acc[8][4];
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        vr += __shfl_xor_sync(FULL, vr, d); pr += __shfl_xor_sync(FULL, pr, d);
        vl += __shfl_xor_sync(FULL, vl, d); pl += __shfl_xor_sync(FULL, pl, d);
    }
    if (lane == 0) { s_acc[wib][0] = vr; s_acc[wib][1] = pr; s_acc[wib][2] = vl; s_acc[wib][3] = pl; }
    __syncthreads();
    if (threadIdx.x < 4) {
        unsigned long long t = 0;
#pragma unroll
        for (int w = 0; w < 8; ++w) t += s_acc[w][threadIdx.x];
        if (t) atomicAdd(&m.ctr->pr_vox_removed + threadIdx.x, t);
    }

    if (last_block_done(&m.ctr->ticket[1]) && threadIdx.x == 0) {
        volatile Counters* c = m.ctr;
        const unsigned long long removed = c->pr_vox_removed, left = c->pr_vox_left;
        if (out) {
            out->n_voxels_removed = (int64_t)removed;
            out->n_points_removed = (int64_t)c->pr_pts_removed;
            out->n_voxels_left = (int64_t)left;
            out->n_points_left = (int64_t)c->pr_pts_left;
        }
        c->pr_vox_removed = 0ull; c->pr_pts_removed = 0ull; c->pr_vox_left = 0ull; c->pr_pts_left = 0ull;
        const unsigned dead = c->n_dead + (unsigned)removed;
        c->n_dead = dead;
        // rebuild when dead keys are no longer a small fraction of the live ones, or the table is running out of keys
        c->rehash_flag = (dead > 0u && (dead >= 32u + (unsigned)(left >> 3) || c->n_keys > m.key_limit - (m.key_limit >> 2))) ? 1u : 0u;
        if (removed) { c->full_flag = 0u; m.mail->full = 0u; }     // buckets are available again
    }
}

// ---- in-place rehash (SURVEY.md:214-216: deletion in open addressing), ONE cooperative kernel.  Pass 1 re-inserts every
// entry that owns a bucket into the empty shadow table (16-byte entries only: buckets stay where they are) and recomputes
// the reach words; a grid-wide barrier; pass 2 copies the shadow table back and empties it again.  The kernel returns at
// once unless prune's epilogue (or far_map_rehash) set the flag: the decision is taken on the device, the launch is
// unconditional.
__global__ void __launch_bounds__(256) rehash_kernel(MapView m) {
    if (!m.ctr->rehash_flag) return;
    unsigned n_moved = 0;
    for (uint32_t s = blockIdx.x * blockDim.x + threadIdx.x; s < m.slots; s += gridDim.x * blockDim.x) {
        const Entry e = m.table[s];
        if (e.key != KEY_EMPTY && e.bucket < BUCKET_PENDING) {
            bool claimed;
            Entry seen;
            const uint32_t t = find_or_claim(m.shadow, m.mask, m.slots, e.key, true, claimed, seen);
            m.shadow[t].bucket = e.bucket;
            atomicOr(&m.shadow[t].cr, entry_count(e.cr));     // the reach bits of slot t may be raised concurrently
            ++n_moved;
        }
    }
    n_moved = __reduce_add_sync(FULL, n_moved);
    if (n_moved && (threadIdx.x & 31) == 0) atomicAdd(&m.ctr->rehash_moved, n_moved);
    // grid-wide barrier between the two passes (cooperative launch: every block is resident).  The arrival counter
    // returns to zero by itself: the last block to LEAVE resets it.
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) {
        atomicAdd(&m.ctr->rehash_barrier, 1u);
        while (ld_volatile(&m.ctr->rehash_barrier) < gridDim.x) __nanosleep(64);
        __threadfence();
    }
    __syncthreads();
    for (uint32_t s0 = blockIdx.x * blockDim.x + (threadIdx.x & ~31u); s0 < m.slots; s0 += gridDim.x * blockDim.x) {
        const uint32_t s = s0 + (threadIdx.x & 31u);
        uint4 ent = make_uint4(0xFFFFFFFFu, 0xFFFFFFFFu, BUCKET_PENDING, 0u);
        if (s < m.slots) {
            uint4* sh = reinterpret_cast<uint4*>(m.shadow + s);
            ent = *sh;
            *reinterpret_cast<uint4*>(m.table + s) = ent;
            *sh = make_uint4(0xFFFFFFFFu, 0xFFFFFFFFu, BUCKET_PENDING, 0u);
        }
        // the occupancy bitmap of the rebuilt table: 32 consecutive slots are one word
        const unsigned word = __ballot_sync(FULL, !(ent.x == 0xFFFFFFFFu && ent.y == 0xFFFFFFFFu));
        if ((threadIdx.x & 31u) == 0) m.occ[s0 >> 5] = word;
    }
    if (last_block_done(&m.ctr->ticket[4]) && threadIdx.x == 0) {
        volatile Counters* c = m.ctr;
        c->n_keys = c->rehash_moved;
        c->rehash_moved = 0u;
        c->n_dead = 0u;
        c->n_rehash = c->n_rehash + 1u;
        c->rehash_barrier = 0u;
        c->rehash_flag = 0u;
    }
}

__global__ void set_rehash_flag_kernel(MapView m) {
    if (threadIdx.x == 0 && blockIdx.x == 0) m.ctr->rehash_flag = 1u;
}

// ---- far_map_renumber (R22): ids -= smallest live id, next_id likewise; order and contents unchanged ---------------
__global__ void __launch_bounds__(256) renumber_min_kernel(MapView m) {
    const uint32_t s = blockIdx.x * blockDim.x + threadIdx.x;
    uint32_t mn = NO_ID;
    if (s < m.slots) {
        const Entry e = m.table[s];
        if (e.key != KEY_EMPTY && e.bucket < BUCKET_PENDING && entry_count(e.cr) > 0)
            mn = m.ids[(size_t)e.bucket * m.cap];             // ids ascend inside a bucket
    }
    mn = __reduce_min_sync(FULL, mn);
    if ((threadIdx.x & 31) == 0 && mn != NO_ID) atomicMin(&m.ctr->min_id, mn);
}

__global__ void __launch_bounds__(256) renumber_apply_kernel(MapView m, unsigned long long offered_at) {
    const uint32_t s = blockIdx.x * blockDim.x + threadIdx.x;
    const uint32_t mn = m.ctr->min_id;
    if (s < m.slots && mn != NO_ID && mn != 0u) {
        const Entry e = m.table[s];
        if (e.key != KEY_EMPTY && e.bucket < BUCKET_PENDING) {
            const uint32_t cnt = entry_count(e.cr);
            for (uint32_t j = 0; j < cnt; ++j) {
                const size_t at = (size_t)e.bucket * m.cap + j;
                const uint32_t id = m.ids[at] - mn;
                m.ids[at] = id;
                m.points[at].w = __uint_as_float(id);
            }
        }
    }
    if (last_block_done(&m.ctr->ticket[3]) && threadIdx.x == 0) {
        volatile Counters* c = m.ctr;
        const unsigned long long sub = (mn == NO_ID) ? c->next_id : (unsigned long long)mn;   // empty map: restart at 0
        c->next_id = c->next_id - sub;
        c->call_first_id = c->call_first_id >= sub ? c->call_first_id - sub : 0ull;
        c->min_id = NO_ID;
        // seqlock towards the host (refresh_id_bound): odd while the record is being written, even = 2 x passes completed
        const uint32_t seq = m.mail->renumber_seq;
        m.mail->renumber_seq = seq + 1u;
        __threadfence_system();
        m.mail->next_id_after_renumber = c->next_id;
        m.mail->offered_at_renumber = offered_at;
        __threadfence_system();
        m.mail->renumber_seq = seq + 2u;
    }
}

// far_map_snapshot_restore: the pinned mailbox follows the restored sticky flag
__global__ void mirror_full_kernel(MapView m) {
    if (blockIdx.x == 0 && threadIdx.x == 0) m.mail->full = *reinterpret_cast<volatile unsigned int*>(&m.ctr->full_flag) ? 1u : 0u;
}

// ---- ASMD density (R17): integer sums over the live voxels near the centre, one division at the end --
__global__ void __launch_bounds__(256) asmd_density_kernel(MapView m, double cx, double cy, double cz, double r2,
                                                            unsigned long long* acc /* [2]: voxels, points */) {
    const uint32_t s = blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long nv = 0, np = 0;
    if (s < m.slots) {
        const Entry e = m.table[s];
        const uint32_t cnt = entry_count(e.cr);
        if (e.key != KEY_EMPTY && e.bucket < BUCKET_PENDING && cnt > 0) {
            int k[3];
            unpack_key(e.key, k);
            const double v = (double)m.voxel;
            const double dx = __dadd_rn(__dmul_rn(__dadd_rn((double)k[0], 0.5), v), -cx);
            const double dy = __dadd_rn(__dmul_rn(__dadd_rn((double)k[1], 0.5), v), -cy);
            const double dz = __dadd_rn(__dmul_rn(__dadd_rn((double)k[2], 0.5), v), -cz);
            const double d2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
            if (d2 <= r2) { nv = 1; np = cnt; }
        }
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) { nv += __shfl_xor_sync(FULL, nv, d); np += __shfl_xor_sync(FULL, np, d); }
    if ((threadIdx.x & 31) == 0 && nv) { atomicAdd(&acc[0], nv); atomicAdd(&acc[1], np); }
}

__global__ void asmd_density_out_kernel(MapView m, unsigned long long* acc, double* out) {
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        out[0] = acc[0] ? __ddiv_rn((double)acc[1], (double)acc[0]) : (double)m.cap;
        out[1] = (double)acc[0];
        acc[0] = 0ull; acc[1] = 0ull;
    }
}

// ---- clear: empty the table, give every used bucket a clean id row, re-arm the counters (one launch) ----------------
__global__ void __launch_bounds__(256) clear_kernel(MapView m) {
    const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x, nthr = gridDim.x * blockDim.x;
    for (uint32_t s = tid; s < m.slots; s += nthr)
        *reinterpret_cast<uint4*>(m.table + s) = make_uint4(0xFFFFFFFFu, 0xFFFFFFFFu, BUCKET_PENDING, 0u);
    for (uint32_t w = tid; w < (m.slots + 31u) / 32u; w += nthr) m.occ[w] = 0u;
    const size_t used = (size_t)min(m.ctr->bump, m.max_buckets) * (size_t)m.cap;   // fresh buckets beyond are clean
    for (size_t j = tid; j < used; j += nthr) m.ids[j] = NO_ID;
    if (last_block_done(&m.ctr->ticket[2]) && threadIdx.x == 0) {
        Counters z;
        memset(&z, 0, sizeof(z));
        z.min_id = NO_ID;
        *m.ctr = z;
        m.mail->full = 0u;
    }
}

__global__ void __launch_bounds__(256) table_init_kernel(Entry* table, uint32_t slots) {
    const uint32_t s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= slots) return;
    *reinterpret_cast<uint4*>(table + s) = make_uint4(0xFFFFFFFFu, 0xFFFFFFFFu, BUCKET_PENDING, 0u);
}

// ---- stats / export ----------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) stats_kernel(MapView m, unsigned long long* acc /* [3] */) {
    const uint32_t s = blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long nv = 0, np = 0, nd = 0;
    if (s < m.slots) {
        const Entry e = m.table[s];
        if (e.key != KEY_EMPTY) {
            const uint32_t cnt = entry_count(e.cr);
            if (e.bucket < BUCKET_PENDING && cnt > 0) { nv = 1; np = cnt; } else nd = 1;
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

__global__ void stats_out_kernel(MapView m, unsigned long long* acc, far_map_stats_t* out) {
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        const Counters* c = m.ctr;
        out->n_voxels = (int64_t)acc[0];
        out->n_points = (int64_t)acc[1];
        out->n_dead_keys = (int64_t)acc[2];
        out->n_slots = (int64_t)m.slots;
        out->next_id = c->next_id;
        out->n_keys = (int64_t)c->n_keys;
        out->n_free_buckets = (int64_t)max(c->n_free, 0);
        out->n_fresh_buckets = (int64_t)m.max_buckets - (int64_t)min(c->bump, m.max_buckets);
        out->n_rehash = (int64_t)c->n_rehash;
        out->full = (int64_t)c->full_flag;
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
    e.key = KEY_EMPTY; e.bucket = NO_BUCKET; e.cr = 0;
    if (s < m.slots) e = m.table[s];
    const uint32_t my_cnt = entry_count(e.cr);
    const bool live = e.key != KEY_EMPTY && e.bucket < BUCKET_PENDING && my_cnt > 0;
    const unsigned b = __ballot_sync(FULL, live);
    if (!b) return;
    unsigned long long base = 0;
    if (lane == 0) base = atomicAdd(n_out, (unsigned long long)__popc(b));
    base = __shfl_sync(FULL, base, 0);
    const unsigned long long row = base + __popc(b & ((1u << lane) - 1u));
    if (live && (int64_t)row < max_out) {
        keys[row] = e.key;
        counts[row] = (int32_t)my_cnt;
    }
    // cooperative copy of each live bucket of this warp
    unsigned rem = b;
    while (rem) {
        const int src = __ffs(rem) - 1;
        rem &= rem - 1;
        const uint32_t bk = __shfl_sync(FULL, e.bucket, src);
        const uint32_t cnt = __shfl_sync(FULL, my_cnt, src);
        const unsigned long long r = __shfl_sync(FULL, row, src);
        if ((int64_t)r >= max_out) continue;
        for (uint32_t j = lane; j < (uint32_t)m.cap; j += 32) {
            const bool have = j < cnt;
            const size_t from = (size_t)bk * m.cap + j, to = (size_t)r * m.cap + j;
            if (pts) pts[to] = have ? m.points[from] : make_float4(0.f, 0.f, 0.f, __uint_as_float(NO_ID));
            if (cov6) {
                for (int a = 0; a < 6; ++a) cov6[to * 6 + a] = (have && m.cov) ? m.cov[from * 6 + a] : 0.f;
            }
            if (cov_ok) cov_ok[to] = (have && m.cov_ok) ? m.cov_ok[from] : 0;
        }
    }
}

__global__ void write_i64_kernel(unsigned long long* src, int64_t* dst) {
    if (threadIdx.x == 0 && blockIdx.x == 0) { *dst = (int64_t)*src; *src = 0ull; }
}

__global__ void __launch_bounds__(256) voxel_keys_kernel(const float* __restrict__ xyz, int64_t n, int stride, float v,
                                                          unsigned long long* __restrict__ keys) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float* p = xyz + i * stride;
    int k[3];
    keys[i] = voxel_index(p[0], p[1], p[2], v, k) ? pack_key(k[0], k[1], k[2]) : KEY_EMPTY;
}

}  // namespace far

// =============================================================================================================
extern "C" {

const char* far_strerror(int status) {
    switch (status) {
        case FAR_OK: return "ok";
        case FAR_ERR_ARG: return "invalid argument";
        case FAR_ERR_CUDA: return "CUDA runtime error";
        case FAR_ERR_FULL: return "voxel map full: points were dropped";
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
    if (!(c.min_spacing >= 0.0)) return FAR_ERR_ARG;
    if (c.renumber_every == 0) c.renumber_every = 1ll << 31;
    if (c.renumber_every < 1 || c.renumber_every > (1ll << 31)) return FAR_ERR_ARG;
    uint64_t slots = 16;
    const double want = (double)c.max_voxels / (double)c.max_load;
    while ((double)slots < want) slots <<= 1;
    if (slots >= (1ull << 31) || (uint64_t)c.max_voxels * (uint64_t)c.cap >= (1ull << 32)) return FAR_ERR_ARG;   // refs are 32-bit

    far_map* m = new (std::nothrow) far_map();
    if (!m) return FAR_ERR_ARG;
    memset(m, 0, sizeof(*m));
    m->cfg = c;
    m->max_batch = c.max_batch;
    m->renumber_every = (uint64_t)c.renumber_every;
    FAR_CUDA(cudaGetDevice(&m->device));
    FAR_CUDA(cudaDeviceGetAttribute(&m->sm_count, cudaDevAttrMultiProcessorCount, m->device));
    FAR_CUDA(cudaDeviceGetAttribute(&m->l2_bytes, cudaDevAttrL2CacheSize, m->device));
    MapView& v = m->view;
    v.slots = (uint32_t)slots;
    v.mask = (uint32_t)slots - 1;
    v.max_buckets = (uint32_t)c.max_voxels;
    v.key_limit = (uint32_t)(slots - slots / 16);
    v.cap = c.cap;
    v.k_cov = c.k_cov;
    v.voxel = c.voxel_size;
    v.cov_eps = c.cov_eps;
    const size_t npts = (size_t)c.max_voxels * c.cap;
    cudaError_t e = cudaSuccess;
    auto alloc = [&](void** p, size_t bytes) { if (e == cudaSuccess) e = cudaMalloc(p, bytes); };
    alloc((void**)&v.table, slots * sizeof(Entry));
    alloc((void**)&v.shadow, slots * sizeof(Entry));
    alloc((void**)&v.points, npts * sizeof(float4));
    alloc((void**)&v.ids, npts * sizeof(uint32_t));
    alloc((void**)&v.free_list, (size_t)c.max_voxels * sizeof(uint32_t));
    alloc((void**)&v.occ, ((slots + 31) / 32) * sizeof(uint32_t));
    if (c.with_cov) {
        alloc((void**)&v.cov, npts * 6 * sizeof(float));
        alloc((void**)&v.cov_ok, npts);
    }
    alloc((void**)&v.ctr, sizeof(Counters));
    v.touched_sub_cap = (uint32_t)((((c.max_batch + 255) / 256 + TOUCHED_SUBS - 1) / TOUCHED_SUBS + 1) * 256);
    alloc((void**)&m->d_touched, (size_t)TOUCHED_SUBS * v.touched_sub_cap * sizeof(uint32_t));
    alloc((void**)&v.touched_cnt, (size_t)TOUCHED_SUBS * 32 * sizeof(uint32_t));
    alloc((void**)&m->d_cov_list, (size_t)c.max_batch * sizeof(uint4));
    if (c.min_spacing > 0.0) {            // scratch of the regular-spacing insert (R21)
        alloc((void**)&m->d_sp_cnt, (size_t)c.max_voxels * sizeof(uint32_t));
        alloc((void**)&m->d_sp_vt, (size_t)c.max_voxels * sizeof(uint32_t));
        alloc((void**)&m->d_sp_ptb, (size_t)c.max_batch * sizeof(uint32_t));
        alloc((void**)&m->d_sp_start, ((size_t)c.max_batch + 1) * sizeof(uint32_t));
        alloc((void**)&m->d_sp_seg, (size_t)c.max_batch * sizeof(uint32_t));
    }
    if (e == cudaSuccess) e = cudaHostAlloc((void**)&m->h_mail, sizeof(Mailbox), cudaHostAllocMapped);
    if (e == cudaSuccess) {
        memset((void*)m->h_mail, 0, sizeof(Mailbox));
        e = cudaHostGetDevicePointer((void**)&v.mail, (void*)m->h_mail, 0);
    }
    if (e != cudaSuccess) {
        far::set_cuda_error(e, "allocation in far_map_create");
        far_map_destroy(m);
        return FAR_ERR_CUDA;
    }
    // empty tables: every key = ~0, no bucket; every id word = FAR_NO_ID
    FAR_CUDA(cudaMemset(v.ids, 0xFF, npts * sizeof(uint32_t)));
    FAR_LAUNCH(table_init_kernel, grid_for((int64_t)slots, 256), 256, 0, 0, v.table, v.slots);
    FAR_LAUNCH(table_init_kernel, grid_for((int64_t)slots, 256), 256, 0, 0, v.shadow, v.slots);
    FAR_CUDA(cudaGetLastError());
    Counters z;
    memset(&z, 0, sizeof(z));
    z.min_id = NO_ID;
    FAR_CUDA(cudaMemcpy(v.ctr, &z, sizeof(z), cudaMemcpyHostToDevice));
    if (v.cov_ok) FAR_CUDA(cudaMemset(v.cov_ok, 0, npts));
    FAR_CUDA(cudaMemset(v.touched_cnt, 0, (size_t)TOUCHED_SUBS * 32 * sizeof(uint32_t)));
    FAR_CUDA(cudaMemset(v.occ, 0, ((slots + 31) / 32) * sizeof(uint32_t)));
    if (m->d_sp_cnt) FAR_CUDA(cudaMemset(m->d_sp_cnt, 0, (size_t)c.max_voxels * sizeof(uint32_t)));
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
    cudaFree(m->view.table); cudaFree(m->view.shadow); cudaFree(m->view.points); cudaFree(m->view.ids);
    cudaFree(m->view.free_list); cudaFree(m->view.occ); cudaFree(m->view.cov); cudaFree(m->view.cov_ok);
    cudaFree(m->view.ctr); cudaFree(m->d_touched); cudaFree(m->view.touched_cnt); cudaFree(m->d_cov_list);
    cudaFree(m->d_gicp_partials);
    cudaFree(m->d_sp_cnt); cudaFree(m->d_sp_vt); cudaFree(m->d_sp_ptb); cudaFree(m->d_sp_start); cudaFree(m->d_sp_seg);
    if (m->h_mail) cudaFreeHost((void*)m->h_mail);
    delete m;
    return FAR_OK;
}

int far_map_clear(far_map_t* m, void* stream) {
    if (!m) return FAR_ERR_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    FAR_LAUNCH(clear_kernel, m->sm_count * 4, 256, 0, st, m->view);
    FAR_CUDA(cudaGetLastError());
    m->next_id_ub = 0;
    m->offered_total = 0;
    m->offered_at_renumber = 0;
    return FAR_OK;
}

// folds a completed renumber pass (reported through the mailbox) into the host-side bound of the id counter
// The mailbox record {next_id_after_renumber, offered_at_renumber} is guarded by a sequence word the device makes odd
// before it writes the record and even (2 x passes completed) after: the host takes a record only if it read the same
// even value before and after the two fields.  Passes enqueued before the last far_map_snapshot_restore describe a counter
// the restore has overwritten: they are marked seen and not folded (the restored bound stays a valid upper bound).
static void refresh_id_bound(far_map_t* m) {
    const uint32_t seq = m->h_mail->renumber_seq;
    if ((seq & 1u) || seq == m->renumber_seen) return;          // a record is being written, or nothing new
    std::atomic_thread_fence(std::memory_order_acquire);
    const uint64_t at = m->h_mail->offered_at_renumber, nid = m->h_mail->next_id_after_renumber;
    std::atomic_thread_fence(std::memory_order_acquire);
    if (m->h_mail->renumber_seq != seq) return;                 // a newer pass is landing: take it next time
    m->renumber_seen = seq;
    if (seq / 2u <= m->renumber_ignore) return;                 // enqueued before the last snapshot restore
    if (at <= m->offered_total) m->next_id_ub = nid + (m->offered_total - at);
}

static int renumber_enqueue(far_map_t* m, cudaStream_t st) {
    FAR_LAUNCH(renumber_min_kernel, grid_for(m->view.slots, 256), 256, 0, st, m->view);
    FAR_LAUNCH(renumber_apply_kernel, grid_for(m->view.slots, 256), 256, 0, st, m->view, (unsigned long long)m->offered_total);
    FAR_CUDA(cudaGetLastError());
    m->offered_at_renumber = m->offered_total;
    m->renumber_enqueued += 1u;
    return FAR_OK;
}

int far_map_renumber(far_map_t* m, void* stream) {
    if (!m) return FAR_ERR_ARG;
    return renumber_enqueue(m, (cudaStream_t)stream);
}

} // extern "C"

// n = min(n, *d_n) if d_n is given (single chunk only: n <= max_batch); the host-side id bound advances by n
int far::insert_impl(far_map_t* m, const float* d_xyz, int64_t n, const int64_t* d_n, int stride, int pose_mode, const far_pose_t* hpose,
                     const far_pose_t* d_pose, int compute_cov, far_insert_stats_t* d_stats, void* stream, const double* d_n_close,
                     double d_max) {
    if (!m || (!d_xyz && n > 0) || n < 0 || n > 0x7FFFFFFFll || (stride != 3 && stride != 4)) return FAR_ERR_ARG;
    Asmd asmd{d_n_close, d_n_close ? d_max : 1.0, d_n_close ? 1 : 0};
    if (d_n && n > m->max_batch) return FAR_ERR_ARG;
    Spaced sp;
    memset(&sp, 0, sizeof(sp));
    if (m->cfg.min_spacing > 0.0) {
        sp.offer_cnt = m->d_sp_cnt; sp.voxel_t = m->d_sp_vt; sp.pt_bucket = m->d_sp_ptb; sp.seg_start = m->d_sp_start; sp.seg = m->d_sp_seg;
        sp.s2 = m->cfg.min_spacing * m->cfg.min_spacing;
        sp.on = 1;
    }
    if (compute_cov && !m->view.cov) return FAR_ERR_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    // id counter (R3: ids are u32 and advance by the points OFFERED).  The counter lives on the device; the host keeps an
    // upper bound, enqueues a renumber pass (R22) at a deterministic point of the offered-points count, and only if the
    // bound would still overflow does it wait for the device to report the renumbered counter.
    refresh_id_bound(m);
    if (m->offered_total - m->offered_at_renumber + (uint64_t)n > m->renumber_every && m->offered_total > m->offered_at_renumber) {
        const int rc = renumber_enqueue(m, st);
        if (rc != FAR_OK) return rc;
    }
    if (m->next_id_ub + (uint64_t)n > 0xFFFFFFFFull) {
        FAR_CUDA(cudaStreamSynchronize(st));
        refresh_id_bound(m);
        if (m->next_id_ub + (uint64_t)n > 0xFFFFFFFFull) return FAR_ERR_RANGE;
    }
    Pose hp;
    memset(&hp, 0, sizeof(hp));
    if (pose_mode == 1) memcpy(&hp, hpose, sizeof(hp));
    const bool cov_by_list = compute_cov && n <= m->max_batch;
    const int commit_grid = m->sm_count * 8;
    int64_t off = 0;
    do {
        const int64_t nc = (n - off < m->max_batch) ? n - off : m->max_batch;
        const float* xyz = d_xyz + off * stride;
        const int last = off + nc >= n;
        if (nc > 0)
            FAR_LAUNCH(insert_claim_chain_kernel, grid_for(nc, 256), 256, 0, st, m->view, xyz, nc, d_n, stride, pose_mode, hp,
                                                                          (const Pose*)d_pose, (uint32_t)off, m->d_touched, asmd, sp);
        if (sp.on) {
            // R21: list -> scan -> scatter -> per-voxel sort and sequential walk (closes the chunk like the commit kernel)
            if (nc > 0) {
                FAR_LAUNCH(spaced_scan_kernel, 1, 1024, 0, st, m->view, m->d_touched, sp);
                FAR_LAUNCH(spaced_scatter_kernel, grid_for(nc, 256), 256, 0, st, m->view, nc, d_n, sp);
            }
            FAR_LAUNCH(spaced_commit_kernel, nc > 0 ? m->sm_count * 8 : 1, SP_THREADS, 0, st, m->view, xyz, nc, stride, pose_mode, hp,
                                                               (const Pose*)d_pose, (uint32_t)off, m->d_touched,
                                                               cov_by_list ? m->d_cov_list : nullptr, n, d_n, last, d_stats, asmd, sp);
        } else
        FAR_LAUNCH(insert_commit_kernel, nc > 0 ? commit_grid : 1, 256, 0, st, m->view, xyz, stride, pose_mode, hp,
                                                           (const Pose*)d_pose, (uint32_t)off, m->d_touched,
                                                           cov_by_list ? m->d_cov_list : nullptr, n, d_n, last, d_stats);
        FAR_CUDA(cudaGetLastError());
        off += nc;
    } while (off < n);
    m->next_id_ub += (uint64_t)n;
    m->offered_total += (uint64_t)n;
    if (compute_cov && n > 0) {
        // "we recompute the covariances of the added points" -- against the map AFTER the insert
        int rc = cov_by_list ? launch_knn_cov_refs(m, m->d_cov_list, &m->view.ctr->n_tasks, n, st)
                              : launch_knn_cov_new_ids(m, st);
        if (rc != FAR_OK) return rc;
    }
    // the device's sticky flag, seen without a synchronisation: set by THIS call only if it has already run
    return m->h_mail->full ? FAR_ERR_FULL : FAR_OK;
}

extern "C" {

int far_map_insert(far_map_t* m, const float* d_xyz, int64_t n, int stride, const far_pose_t* pose, int compute_cov,
                   far_insert_stats_t* d_stats, void* stream) {
    return far::insert_impl(m, d_xyz, n, nullptr, stride, pose ? 1 : 0, pose, nullptr, compute_cov, d_stats, stream, nullptr, 1.0);
}

int far_map_insert_dev(far_map_t* m, const float* d_xyz, int64_t n, int stride, const far_pose_t* d_pose,
                       int compute_cov, far_insert_stats_t* d_stats, void* stream) {
    if (!d_pose) return FAR_ERR_ARG;
    return far::insert_impl(m, d_xyz, n, nullptr, stride, 2, nullptr, d_pose, compute_cov, d_stats, stream, nullptr, 1.0);
}

int far_map_insert_asmd(far_map_t* m, const float* d_xyz, int64_t n, int stride, const far_pose_t* pose,
                        const double* d_n_close, double d_max, int compute_cov, far_insert_stats_t* d_stats, void* stream) {
    if (!d_n_close || !(d_max > 0.0)) return FAR_ERR_ARG;
    return far::insert_impl(m, d_xyz, n, nullptr, stride, pose ? 1 : 0, pose, nullptr, compute_cov, d_stats, stream, d_n_close, d_max);
}

int far_map_insert_asmd_dev(far_map_t* m, const float* d_xyz, int64_t n, int stride, const far_pose_t* d_pose,
                            const double* d_n_close, double d_max, int compute_cov, far_insert_stats_t* d_stats,
                            void* stream) {
    if (!d_pose || !d_n_close || !(d_max > 0.0)) return FAR_ERR_ARG;
    return far::insert_impl(m, d_xyz, n, nullptr, stride, 2, nullptr, d_pose, compute_cov, d_stats, stream, d_n_close, d_max);
}

// PAPER.md:109 "the average amount of points per voxel in a close range of the current scan" (R17)
int far_asmd_density(const far_map_t* local, const double center[3], double r_close, double* d_out, void* stream) {
    if (!local || !center || !d_out || !(r_close >= 0.0)) return FAR_ERR_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    unsigned long long* acc = local->view.ctr->scratch + 4;     // two words, left zeroed by the out kernel
    FAR_LAUNCH(asmd_density_kernel, grid_for(local->view.slots, 256), 256, 0, st, local->view, center[0], center[1], center[2],
                                                                        r_close * r_close, acc);
    FAR_LAUNCH(asmd_density_out_kernel, 1, 32, 0, st, local->view, acc, d_out);
    FAR_CUDA(cudaGetLastError());
    return FAR_OK;
}

static int rehash_enqueue(far_map_t* m, cudaStream_t st) {
    // grid-stride over the table with one resident wave: when the flag is clear (most frames) the launch costs a few
    // hundred empty blocks, not one per 256 slots
    // ONE cooperative launch (the two passes are separated by a grid-wide barrier inside the kernel), sized to a resident
    // wave: when the flag is clear (most frames) it costs a few hundred blocks that return at once
    static int per_sm = 0;
    if (per_sm == 0) {
        int v = 0;
        FAR_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&v, rehash_kernel, 256, 0));
        per_sm = v < 1 ? 1 : v;
    }
    int grid = grid_for(m->view.slots, 256);
    if (grid > m->sm_count * per_sm) grid = m->sm_count * per_sm;
    MapView view = m->view;
    void* args[] = {(void*)&view};
    {
        far::LaunchScope ls_("rehash_kernel", st);
        FAR_CUDA(cudaLaunchCooperativeKernel((const void*)rehash_kernel, dim3((unsigned)grid), dim3(256), args, 0, st));
    }
    return FAR_OK;
}

static int prune_impl(far_map_t* m, const double* c, const far_pose_t* d_pose, double radius, far_prune_stats_t* d_stats,
                      void* stream) {
    if (!m || (!c && !d_pose)) return FAR_ERR_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    const double r2 = radius * radius;
    FAR_LAUNCH(prune_kernel, std::min(grid_for(m->view.slots, 256 * 4), m->sm_count * 8), 256, 0, st, m->view, c ? c[0] : 0.0, c ? c[1] : 0.0, c ? c[2] : 0.0,
                                                                (const Pose*)d_pose, r2, d_stats);
    FAR_CUDA(cudaGetLastError());
    return rehash_enqueue(m, st);          // returns at once unless prune's epilogue asked for the rebuild
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
    unsigned long long* acc = m->view.ctr->scratch;
    FAR_LAUNCH(stats_kernel, grid_for(m->view.slots, 256), 256, 0, st, m->view, acc);
    FAR_LAUNCH(stats_out_kernel, 1, 32, 0, st, m->view, acc, d_stats);
    FAR_CUDA(cudaGetLastError());
    return FAR_OK;
}

int far_map_status(const far_map_t* m) {
    if (!m) return FAR_ERR_ARG;
    return m->h_mail->full ? FAR_ERR_FULL : FAR_OK;
}

int far_map_export(far_map_t* m, uint64_t* d_keys, int32_t* d_counts, float* d_points4, float* d_cov6,
                   uint8_t* d_cov_valid, int64_t max_out, int64_t* d_n_voxels, void* stream) {
    if (!m || !d_keys || !d_counts || !d_n_voxels || max_out < 0) return FAR_ERR_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    unsigned long long* acc = m->view.ctr->scratch + 3;          // left zeroed by write_i64_kernel
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

// Drops the dead keys now, whatever their number: two stream-ordered launches, no allocation, no synchronisation.
// far_map_prune does the same by itself whenever the dead keys pass its threshold.
int far_map_rehash(far_map_t* m, void* stream) {
    if (!m) return FAR_ERR_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    FAR_LAUNCH(set_rehash_flag_kernel, 1, 32, 0, st, m->view);
    return rehash_enqueue(m, st);
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

long long launch_counter() { return g_launches.load(std::memory_order_relaxed); }
void launch_counter_add(long long n) { g_launches.fetch_add(n, std::memory_order_relaxed); }
bool profiling_enabled() { return g_prof.load(std::memory_order_relaxed) != 0; }

LaunchScope::~LaunchScope() {
    if (rec_ >= 0) {
        std::lock_guard<std::mutex> lk(g_prof_mu);
        cudaEventRecord(g_recs[rec_].b, st_);
    }
}

}  // namespace far

struct far_snapshot {
    void *table, *points, *ids, *cov, *cov_ok, *free_list, *ctr, *occ;
    size_t b_table, b_points, b_ids, b_cov, b_ok, b_free, b_occ;
    uint64_t next_id_ub, offered_total, offered_at_renumber;
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
    cudaFree(s->table); cudaFree(s->points); cudaFree(s->ids); cudaFree(s->cov); cudaFree(s->cov_ok); cudaFree(s->free_list);
    cudaFree(s->ctr); cudaFree(s->occ);
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
    const size_t npts = (size_t)m->view.max_buckets * m->view.cap;
    s->b_table = (size_t)m->view.slots * sizeof(Entry);
    s->b_points = npts * sizeof(float4);
    s->b_ids = npts * sizeof(uint32_t);
    s->b_cov = m->view.cov ? npts * 6 * sizeof(float) : 0;
    s->b_ok = m->view.cov_ok ? npts : 0;
    s->b_free = (size_t)m->view.max_buckets * sizeof(uint32_t);
    s->b_occ = (((size_t)m->view.slots + 31) / 32) * sizeof(uint32_t);
    s->next_id_ub = m->next_id_ub;
    s->offered_total = m->offered_total;
    s->offered_at_renumber = m->offered_at_renumber;
    struct { void** dst; const void* src; size_t bytes; } parts[] = {
        {&s->table, m->view.table, s->b_table}, {&s->points, m->view.points, s->b_points}, {&s->ids, m->view.ids, s->b_ids},
        {&s->cov, m->view.cov, s->b_cov}, {&s->cov_ok, m->view.cov_ok, s->b_ok}, {&s->free_list, m->view.free_list, s->b_free},
        {&s->ctr, m->view.ctr, sizeof(Counters)}, {&s->occ, m->view.occ, s->b_occ}};
    cudaError_t e = cudaSuccess;
    for (auto& p : parts) {
        if (!p.bytes || e != cudaSuccess) continue;
        e = cudaMalloc(p.dst, p.bytes);
        if (e == cudaSuccess) e = cudaMemcpyAsync(*p.dst, p.src, p.bytes, cudaMemcpyDeviceToDevice, st);
    }
    if (e != cudaSuccess) {
        far::set_cuda_error(e, "far_map_snapshot_create");
        far_map_snapshot_destroy(s);
        return FAR_ERR_CUDA;
    }
    *out = s;
    return FAR_OK;
}

// the shadow table is empty between calls and the GICP scratch carries its own launch sequence: neither is part of a snapshot
int far_map_snapshot_restore(far_map_t* m, const far_snapshot_t* s, void* stream) {
    if (!m || !s) return FAR_ERR_ARG;
    const size_t npts = (size_t)m->view.max_buckets * m->view.cap;
    if (s->b_table != (size_t)m->view.slots * sizeof(Entry) || s->b_points != npts * sizeof(float4)) return FAR_ERR_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    FAR_CUDA(cudaMemcpyAsync(m->view.table, s->table, s->b_table, cudaMemcpyDeviceToDevice, st));
    FAR_CUDA(cudaMemcpyAsync(m->view.points, s->points, s->b_points, cudaMemcpyDeviceToDevice, st));
    FAR_CUDA(cudaMemcpyAsync(m->view.ids, s->ids, s->b_ids, cudaMemcpyDeviceToDevice, st));
    if (s->b_cov && m->view.cov) FAR_CUDA(cudaMemcpyAsync(m->view.cov, s->cov, s->b_cov, cudaMemcpyDeviceToDevice, st));
    if (s->b_ok && m->view.cov_ok) FAR_CUDA(cudaMemcpyAsync(m->view.cov_ok, s->cov_ok, s->b_ok, cudaMemcpyDeviceToDevice, st));
    FAR_CUDA(cudaMemcpyAsync(m->view.free_list, s->free_list, s->b_free, cudaMemcpyDeviceToDevice, st));
    FAR_CUDA(cudaMemcpyAsync(m->view.ctr, s->ctr, sizeof(Counters), cudaMemcpyDeviceToDevice, st));
    FAR_CUDA(cudaMemcpyAsync(m->view.occ, s->occ, s->b_occ, cudaMemcpyDeviceToDevice, st));
    // the host-visible mirror of the sticky full flag follows the restored counters (a map that filled up after the snapshot
    // would otherwise keep answering FAR_ERR_FULL), and renumber passes enqueued so far no longer describe this counter
    FAR_LAUNCH(mirror_full_kernel, 1, 32, 0, st, m->view);
    FAR_CUDA(cudaGetLastError());
    m->renumber_ignore = m->renumber_enqueued;
    m->next_id_ub = s->next_id_ub;
    m->offered_total = s->offered_total;
    m->offered_at_renumber = s->offered_at_renumber;
    return FAR_OK;
}

}  // extern "C"
