/*
 * far.h -- C ABI of the B200-native FAR-LIO front-end hot path (voxel hashmap + sparsity-aware GICP).
 *
 * Source of the method: /root/reference/PAPER.md (FAR-LIO, arxiv/paper_2606_26010), cited below as
 * PAPER.md:<line>.  Readings of passages the paper leaves open are numbered R1..R22 in DESIGN.md.
 * Every entry point below runs hand-written CUDA kernels for sm_100a; there is no CPU fallback.
 *
 * Conventions
 *  - Every function returns an int status (FAR_OK = 0).  No exception crosses the ABI.
 *  - Pointers named d_* and all bulk arrays (points, ids, covariances, result structs) are DEVICE pointers
 *    (or any device-accessible pointer such as pinned mapped host memory) owned by the caller; the library
 *    never frees, reallocates or retains them beyond the call's stream order.
 *  - Small POD inputs (far_map_config_t, far_pose_t, far_gicp_options_t, prune centre) are HOST pointers,
 *    read during the call.  The *_dev variants read a pose from a DEVICE pointer in stream order, so a frame
 *    pipeline (register -> insert -> prune) needs no host synchronisation.
 *  - `stream` is a cudaStream_t passed as void*.  Calls enqueue work and return; nothing synchronises
 *    unless stated.  The map handle owns all of its device memory, allocated once in far_map_create
 *    (preallocate; allocation spikes show up as latency peaks).
 *  - Points are fp32, `stride` floats apart (3 or 4).  Non-finite points and points whose voxel index leaves
 *    +-2^20 are skipped and counted as invalid.  Poses are map_from_sensor, R row-major, FP64.
 *  - A map handle is not thread-safe; calls on one map must be issued in one stream order.
 */
#ifndef FAR_H
#define FAR_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

enum {
    FAR_OK = 0,
    FAR_ERR_ARG = 1,        /* null pointer, bad stride/size/config */
    FAR_ERR_CUDA = 2,       /* a CUDA runtime call failed (see far_last_cuda_error) */
    FAR_ERR_FULL = 3,       /* the map's bucket pool (max_voxels) or key table is exhausted: points that would open a NEW
                               voxel were dropped and counted.  The condition is raised on the device; far_map_insert*,
                               far_frontend_process* and far_map_status report it from a flag the device mirrors into
                               pinned host memory, i.e. WITHOUT a synchronisation: a call returns it once the kernels of
                               an earlier call (or, after a sync, its own) have dropped points.  The call that returns
                               it has still enqueued all of its work; the flag clears when a prune frees buckets or
                               the map is cleared */
    FAR_ERR_RANGE = 4,      /* id counter would exceed 2^32-1 even after renumbering */
    FAR_ERR_DEGENERATE = 5  /* fewer than 6 inliers or H not positive definite; pose returned = init pose */
};

enum { FAR_KERNEL_CAUCHY = 0, FAR_KERNEL_GEMAN_MCCLURE = 1, FAR_KERNEL_NONE = 2 };

#define FAR_NO_ID 0xFFFFFFFFu

typedef struct { double R[9]; double t[3]; } far_pose_t;

typedef struct {
    float voxel_size;      /* v > 0 [m]                      PAPER.md:62,68 (paper: 4 m)                  */
    int32_t cap;           /* max points per voxel, 1..64    PAPER.md:62,68 (paper: N_max = 40)           */
    int64_t max_voxels;    /* buckets in the dense pool = live voxels the map can hold (exact limit)       */
    float max_load;        /* table load limit in (0,0.9]; 0 -> 0.5; slots = pow2 >= max_voxels / max_load */
    int32_t with_cov;      /* 1: allocate per-point covariance storage (needed for GICP targets)           */
    int32_t k_cov;         /* neighbours for Eq. 1; 0 -> 10                                   */
    double cov_eps;        /* regulariser of Eq. 1; 0 -> 1e-3                                 */
    int64_t max_batch;     /* points per internal insert pass; 0 -> 1<<20.  Larger calls are chunked      */
    int64_t renumber_every;/* offered points between automatic id renumber passes (R22); 0 -> 2^31         */
    double min_spacing;    /* > 0: regular spacing ("regularly spaced ... ~65 cm" at v = 4 m, N_max = 40,
                              i.e. v / sqrt(N_max); R21): an offered point is stored only if no point already stored in
                              ITS OWN voxel is closer (FP64 d2 of R6, strict <), decided in index order after the cap /
                              N_ASMD test.  0: the plain capped insert */
} far_map_config_t;

typedef struct { int64_t n_offered, n_accepted, n_new_voxels, n_dropped_full, n_invalid; } far_insert_stats_t;
typedef struct { int64_t n_voxels_removed, n_points_removed, n_voxels_left, n_points_left; } far_prune_stats_t;
typedef struct {
    int64_t n_voxels, n_points;   /* live voxels and the points stored in them                                       */
    int64_t n_dead_keys;          /* keys of pruned voxels still in the table (dropped by the next rehash)           */
    int64_t n_slots;
    uint64_t next_id;             /* the device-resident id counter                                                  */
    int64_t n_keys;               /* claimed table slots (live + dead)                                               */
    int64_t n_free_buckets;       /* buckets on the free list (returned by prune)                                    */
    int64_t n_fresh_buckets;      /* buckets never used yet                                                          */
    int64_t n_rehash;             /* in-place rehashes since create / clear                                          */
    int64_t full;                 /* 1: points were dropped since buckets were last freed (see FAR_ERR_FULL)         */
} far_map_stats_t;

typedef struct {
    int32_t kernel;      /* FAR_KERNEL_*; Cauchy is the paper's (Eq. 5)       */
    double conv_eps;     /* stop when ||delta||_2 <= conv_eps (5e-3; R13)       */
    double tau_mult;     /* correspondence gate tau = tau_mult * sigma  (R10: 3)              */
    double kappa_div;    /* kernel scale kappa = sigma / kappa_div      (R10: 3)              */
} far_gicp_options_t;

typedef struct {
    far_pose_t pose;     /* registered pose (init pose if status == FAR_ERR_DEGENERATE)                 */
    double H[36];        /* row-major 6x6, order (rho_x,rho_y,rho_z,phi_x,phi_y,phi_z), of the LAST      */
    double b[6];         /*   linearisation performed (at the pose before the final update)              */
    double chi2;         /* sum w * d^T M d of that linearisation                                        */
    int32_t n_inliers, iters, converged, status;
} far_gicp_result_t;

typedef struct far_map far_map_t;
typedef struct far_threshold far_threshold_t;

const char* far_strerror(int status);
/* text of the last CUDA error seen by this library in the calling process ("" if none) */
const char* far_last_cuda_error(void);
/* Tracing: number of kernels this library has launched in the process; optional per-kernel timing with CUDA
 * events on the launching stream.  far_profile_collect synchronises the device, writes one row per kernel name
 * (names are static strings) and clears the records; returns the number of rows. */
long long far_launch_count(void);
void far_profile_enable(int on);
int far_profile_collect(const char** names, double* total_ms, long long* launches, int max_entries);
void far_gicp_default_options(far_gicp_options_t* out);

/* ---- voxel hashmap: PAPER.md:62-68 (cuVoxelMap, Fig. 3), :109 (local submap) -------------------------
 * Open addressing with linear probing on packed 64-bit voxel keys (R1: k = floor(fp32 p / fp32 v), three
 * 21-bit biased indices); 16-byte table entries {key, bucket, count}; buckets of `cap` float4 (x,y,z,id bits) in a dense
 * pool of max_voxels buckets (bump allocator + free list refilled by far_map_prune).
 * far_map_create allocates and initialises all device memory on the current device and synchronises. */
int far_map_create(far_map_t** out, const far_map_config_t* cfg);
int far_map_destroy(far_map_t* map);
/* empties the map and resets the id counter to 0 */
int far_map_clear(far_map_t* map, void* stream);

/* A3/A4 (PAPER.md:62 "fixed, maximum number N_max of points", :109; R3/R4): offers n points.  Point i gets
 * id = next_id + i (next_id advances by n regardless of acceptance).  With a pose the point is first moved in
 * FP64 (fixed operation order, rounded once to fp32).  Result is that of inserting the points one by one in
 * index order: a voxel keeps the lowest ids up to `cap`, in ascending id; batch-invariant and deterministic.
 * compute_cov != 0 (map created with_cov): the covariance (Eq. 1) of every ACCEPTED point is computed against
 * the map after the insert; points already stored keep theirs.
 * d_stats (nullable, device) is overwritten with the totals of this call.
 * Returns FAR_ERR_RANGE (nothing inserted) if the id counter cannot take n more ids, FAR_ERR_FULL (work enqueued) as
 * described at the enum; the exact drop count of this call is d_stats->n_dropped_full.  Two launches per max_batch
 * chunk (+ one for the covariances, served voxel by voxel from a task list the commit kernel leaves); this call itself does not synchronise. */
int far_map_insert(far_map_t* map, const float* d_xyz, int64_t n, int stride, const far_pose_t* pose_or_null,
                   int compute_cov, far_insert_stats_t* d_stats, void* stream);
int far_map_insert_dev(far_map_t* map, const float* d_xyz, int64_t n, int stride, const far_pose_t* d_pose,
                       int compute_cov, far_insert_stats_t* d_stats, void* stream);

/* A5 ("voxels whose distance to the current pose exceeds a certain limit are removed"; R5):
 * removes voxel k iff |(k + 0.5) v - c|^2 > radius^2 (FP64, strict).  centre: HOST double[3]. */
int far_map_prune(far_map_t* map, const double center[3], double radius, far_prune_stats_t* d_stats, void* stream);
/* same, centre = d_pose->t read on the device in stream order */
int far_map_prune_dev(far_map_t* map, const far_pose_t* d_pose, double radius, far_prune_stats_t* d_stats,
                      void* stream);

/* counts live voxels / stored points / dead (pruned) keys and reports the allocator's state (device struct) */
int far_map_stats(far_map_t* map, far_map_stats_t* d_stats, void* stream);
/* FAR_OK or FAR_ERR_FULL from the host-visible mirror of the device's sticky flag; never synchronises */
int far_map_status(const far_map_t* map);
/* Deletion in open addressing (SURVEY.md:214-216; PAPER.md:109 prunes every frame, :171,186 nothing may allocate):
 * far_map_prune hands the buckets of removed voxels back to the free list at once and leaves their keys behind as dead
 * keys; when these pass max(32 + live/8) -- decided on the device in prune's epilogue -- the rehash kernel that
 * every prune call enqueues rebuilds the 16-byte entries into the preallocated shadow table, recomputes the probe bounds and
 * copies them back.  far_map_rehash forces that rebuild now.  No allocation, no synchronisation; contents unchanged. */
int far_map_rehash(far_map_t* map, void* stream);
/* R22 (ids are this library's construct, PAPER.md has none): ids are u32 and advance by the points OFFERED, so a frontend
 * fed 150k-point scans at 20 Hz would exhaust them in ~20 minutes.  A renumber pass subtracts the smallest live id from
 * every stored id and from the id counter (order, contents and every (d2, id) comparison are unchanged).  far_map_insert*
 * enqueues one by itself before the call that would pass `renumber_every` offered points since the last pass; the
 * device reports the new counter through pinned host memory, so the host-side range check needs no synchronisation
 * unless two passes would overlap.  Two stream-ordered launches. */
int far_map_renumber(far_map_t* map, void* stream);

/* Checkpoint / restore of a map's whole device state (table, bucket pool, free list, covariances, counters).
 * create allocates the copy (a maintenance call); restore is eight stream-ordered device copies, no sync. */
typedef struct far_snapshot far_snapshot_t;
int far_map_snapshot_create(far_map_t* map, far_snapshot_t** out, void* stream);
int far_map_snapshot_restore(far_map_t* map, const far_snapshot_t* snap, void* stream);
int far_map_snapshot_destroy(far_snapshot_t* snap);

/* Writes the live voxels in unspecified order: keys[v], counts[v], points4[(v*cap + j)*4 + {0,1,2,3}] =
 * x,y,z,id bits (unused entries 0,0,0,FAR_NO_ID), cov6[(v*cap + j)*6] (xx,xy,xz,yy,yz,zz; nullable),
 * cov_valid[v*cap + j] (nullable).  At most max_out voxels are written; *d_n_voxels = number of live voxels. */
int far_map_export(far_map_t* map, uint64_t* d_keys, int32_t* d_counts, float* d_points4, float* d_cov6,
                   uint8_t* d_cov_valid, int64_t max_out, int64_t* d_n_voxels, void* stream);

/* A1: keys[i] = packed voxel key of point i, ~0 if invalid */
int far_voxel_keys(const float* d_xyz, int64_t n, int stride, float voxel, uint64_t* d_keys, void* stream);

/* A6 ("the voxel containing it as well as all surrounding ones (27 in total)", :80 "closest
 * Euclidean neighbor"; R6): nearest stored point among the 27 voxels around each query by (d^2, id)
 * lexicographic order, d^2 evaluated in FP64 with fixed operation order.  d_id[i] = FAR_NO_ID and
 * d_d2[i] = +inf if no candidate.  d_d2 is the FP64 value rounded to fp32. */
int far_map_nn(const far_map_t* map, const float* d_q, int64_t m, int stride, uint32_t* d_id, float* d_d2,
               void* stream);

/* A7 (Eq. 1; R7/R8): covariance from the k_cov nearest stored points of each query:
 * Sigma_hat (1/k, about the mean), C = Sigma_hat + eps I, Sigma = ||C^-1||_F C.  Fewer than k_cov candidates:
 * valid = 0 and cov6 = identity.  cov6: m*6 fp32 (xx,xy,xz,yy,yz,zz). */
int far_map_knn_cov(const far_map_t* map, const float* d_q, int64_t m, int stride, float* d_cov6,
                    uint8_t* d_valid, void* stream);

/* number of candidate points in the 27 voxels around each query (what A6/A7 scan) and, if d_voxels is not NULL, how many
 * of the 27 voxels are occupied: density probe, used by bench.py for the algorithmic-byte count (27 keys +
 * 4 B per occupied voxel + 16 B per candidate) */
int far_map_count27(const far_map_t* map, const float* d_q, int64_t m, int stride, int32_t* d_count, int32_t* d_voxels,
                    void* stream);

/* A2 ("preprocessing (typically ... deskewing and downsampling)"; R2): one representative per
 * occupied voxel of the scan = the lowest-index valid point, emitted in ascending source index.
 * d_out_xyz: n*3 fp32, d_out_index: n int32, *d_n_out: count.  Call with d_workspace == NULL to get the
 * required workspace size in *workspace_bytes; otherwise *workspace_bytes is the size provided. */
int far_voxelize(const float* d_xyz, int64_t n, int stride, float voxel, float* d_out_xyz, int32_t* d_out_index,
                 int64_t* d_n_out, void* d_workspace, size_t* workspace_bytes, void* stream);

/* far_voxelize for callers that must not allocate device memory: same operation (A2, R2), same outputs bit for bit,
 * but with no workspace argument and no allocation of any kind inside the call (no cudaMalloc / cudaFree, no pool, no
 * allocating library routine -- only a cudaMemsetAsync and the four kernel launches of far_voxelize).
 *
 * Who this is for.  far_voxelize needs about 28 bytes of scratch per point (a throw-away hash table of the scan's voxels,
 * one slot word per point, the tile offsets), and asks the caller to size and provide it.  Some callers cannot: a
 * LiDAR callback that runs inside a hard real-time loop may not call cudaMalloc at all, because the call takes
 * driver-wide locks and can synchronise the whole device for an unbounded time; a component that lives inside
 * somebody else's process (a plug-in of a perception stack, a node whose GPU memory budget was handed out at start-up
 * by a supervisor) often receives its input and output buffers from the host application and has no allocator it is
 * allowed to use; and glue code written in a language binding may have no way to keep a device buffer alive between
 * calls.  For them the scratch lives INSIDE the library, in a file-scope `static __device__` array of
 * FAR_VOXELIZE_STATIC_BYTES bytes (7,341,568 B, about 7 MiB) that every GPU that loads libfar.so carries from the
 * moment the module is loaded on it until the process exits, whether or not this function is ever called.
 *
 * Limit.  n <= FAR_VOXELIZE_STATIC_MAX_POINTS (262,144: two 64 x 2,048 scans, or the three 60k-point racing LiDARs
 * of BASELINE configs[2]).  A larger n is refused with FAR_ERR_ARG before anything is enqueued, and
 * far_last_cuda_error() then names the limit; use far_voxelize with your own workspace for larger scans.
 *
 * First call on a device.  The address of the array is looked up once per device (cudaGetSymbolAddress, with that
 * device current) the first time this function is called while that device is current, and cached.  The look-up is a
 * host-side query, not an allocation, but it may initialise the CUDA context and load the module: make this first call
 * (n = 0 is enough) during set-up, on each device you will use, before the latency-critical part of your program and
 * before any stream capture is begun.  Later calls only enqueue work on `stream`.  At most 64 devices.
 *
 * Sharing.  There is ONE array per device and every call on that device uses it.  It keeps whatever the previous call
 * left in it; the function resets the parts that have to start clean (hash keys and first-index words) on `stream` at
 * the start of every call, so back-to-back calls in one stream are correct.  Two calls whose work can overlap on the
 * same GPU (different streams without an event between them, or two host threads) race on the scratch and produce
 * garbage silently: serialise them, or use far_voxelize with separate workspaces.
 *
 * d_xyz, d_out_xyz, d_out_index, d_n_out: DEVICE pointers owned by the caller, as in far_voxelize (d_out_xyz n*3 fp32,
 * d_out_index n int32, *d_n_out the count).  FAR_ERR_CUDA if the address look-up or a launch fails. */
#define FAR_VOXELIZE_STATIC_MAX_POINTS 262144
#define FAR_VOXELIZE_STATIC_BYTES 7341568
int far_voxelize_static(const float* d_xyz, int64_t n, int stride, float voxel, float* d_out_xyz, int32_t* d_out_index,
                        int64_t* d_n_out, void* stream);

/* A8-A10 (Eq. 2-6; R9-R14).  scan: n source points in the sensor frame with their covariances
 * (d_scan_cov6 n*6 fp32, d_scan_valid n bytes; both nullable = all invalid -> point-to-point).
 * sigma is the adaptive threshold of [1]: gate tau = tau_mult*sigma, kappa = sigma/kappa_div.
 * linearize: one pass at `pose` -> H, b, chi2, n_inliers (pose copied to out, iters = 1).
 * register: Gauss-Newton, T <- Exp(delta) T with H delta = -b, until ||delta|| <= conv_eps or max_iters;
 * the whole loop runs in one cooperative kernel, no host synchronisation inside.  d_out: device-accessible.
 * The map is read-only for the registration, but its handle carries the kernel's reduction scratch and launch sequence:
 * registrations on ONE map must be issued in one stream order (two in flight at once are undefined); registrations on
 * different maps are independent. */
int far_gicp_linearize(const far_map_t* map, const float* d_scan, const float* d_scan_cov6,
                       const uint8_t* d_scan_valid, int64_t n, int stride, const far_pose_t* pose, double sigma,
                       const far_gicp_options_t* opts_or_null, far_gicp_result_t* d_out, void* stream);
int far_gicp_register(const far_map_t* map, const float* d_scan, const float* d_scan_cov6,
                      const uint8_t* d_scan_valid, int64_t n, int stride, const far_pose_t* init_pose,
                      double sigma, int max_iters, const far_gicp_options_t* opts_or_null,
                      far_gicp_result_t* d_out, void* stream);
/* same with n and the initial pose read from DEVICE memory in stream order (n <= n_max rows are allocated) */
int far_gicp_register_dev(const far_map_t* map, const float* d_scan, const float* d_scan_cov6,
                          const uint8_t* d_scan_valid, const int64_t* d_n, int64_t n_max, int stride,
                          const far_pose_t* d_init_pose, double sigma, int max_iters,
                          const far_gicp_options_t* opts_or_null, far_gicp_result_t* d_out, void* stream);
/* same with only n read from DEVICE memory; the initial pose is a HOST pointer passed as a kernel argument (what
 * far_frontend_process uses: the predicted pose comes from the host-side EKF, the scan size from far_voxelize) */
int far_gicp_register_dn(const far_map_t* map, const float* d_scan, const float* d_scan_cov6,
                         const uint8_t* d_scan_valid, const int64_t* d_n, int64_t n_max, int stride,
                         const far_pose_t* init_pose, double sigma, int max_iters,
                         const far_gicp_options_t* opts_or_null, far_gicp_result_t* d_out, void* stream);
/* same as far_map_knn_cov with the query count read from DEVICE memory (for chaining after far_voxelize) */
int far_map_knn_cov_dev(const far_map_t* map, const float* d_q, const int64_t* d_m, int64_t m_max, int stride,
                        float* d_cov6, uint8_t* d_valid, void* stream);

/* ---- motion undistortion ("Preprocessing & Undistortion"; R15/R16) -----------------
 * "the distortion of the LiDAR scan is corrected using the velocity history of the Sensor Fusion.  We perform a
 * linear regression on both the linear and angular velocities ...  This continuous motion model is evaluated in
 * CUDA ... each raw point is undistorted and projected to the frame reference timestamp, which is equal to the
 * scan's final point-timestamp."
 * far_motion_t: body twist xi(t) = a + b (t - t_ref), 6-vectors (linear velocity [m/s] first, then angular
 * velocity [rad/s]), t_ref = frame reference time. */
typedef struct { double a[6]; double b[6]; } far_motion_t;
/* R15, HOST-only FP64 helper (a 6-component line fit, boundary logic): ordinary least squares over m history
 * samples (times[j], vel6[6 j .. 6 j + 5]), all HOST pointers.  Fewer than two distinct times: b = 0, a = mean. */
int far_motion_fit(const double* times, const double* vel6, int32_t m, double t_ref, far_motion_t* out);
/* R16: point i was measured at t_first + d_time[i] (fp32 offsets, DEVICE); Delta_i = dt_ref - (double)d_time[i]
 * with dt_ref = t_ref - t_first (the sweep duration when t_ref is the last point's time).
 *   Omega_i = a Delta_i - b Delta_i^2/2 + [a,b] Delta_i^3/12      (Magnus expansion of the linear twist to second
 *                                                                  order; [.,.] the se(3) bracket)
 *   d_out_xyz[i] = fl32(Exp(-Omega_i) p_i)                        (SE(3) exponential of R12), FP64 arithmetic.
 * motion: HOST pointer, read during the call.  d_out_xyz: n*3 fp32, may NOT alias d_xyz.  Points with a non-finite
 * coordinate or time are copied unchanged.  One pass, 16 B read (28 B at stride 4 with .w) + 12 B written a point. */
int far_undistort(const float* d_xyz, const float* d_time, int64_t n, int stride, double dt_ref,
                  const far_motion_t* motion, float* d_out_xyz, void* stream);

/* ---- Adaptive Submap Density (R17) ------------------------------------------------
 * "Before the map is updated, the average amount of points per voxel in a close range of the current scan is
 * computed ...  we use a linear decay (with a lower bound defined by the k = 10 points required to compute the
 * covariances) ... integrated into the corresponding voxels ... as long as the number of points inside it is
 * below N_ASMD."
 * far_asmd_density: d_out[0] = n_close = mean stored points per live voxel of `local` (the scan-local map of R8)
 * over the voxels with |(k + 0.5) v - center|^2 <= r_close^2 (FP64, R5 form); = cap of `local` if there is none.
 * d_out[1] = number of such voxels (as a double).  center: HOST double[3].  d_out: DEVICE double[2]. */
int far_asmd_density(const far_map_t* local, const double center[3], double r_close, double* d_out, void* stream);
/* far_map_insert with the per-voxel limit
 *   N_ASMD(k) = clamp(floor(n_close (1 - d/d_max) + 0.5), k_cov, cap),  d = |(k + 0.5) v - c|,
 * c = the pose translation (the origin without a pose), every operation one rounded binary64 operation; n_close is
 * read from DEVICE memory (d_n_close[0], e.g. written by far_asmd_density) in stream order.  Same sequential
 * semantics as far_map_insert (R3) with `count < N_ASMD(k)` as the acceptance test; points already stored are never
 * removed, whatever the limit of their voxel has become. */
int far_map_insert_asmd(far_map_t* map, const float* d_xyz, int64_t n, int stride, const far_pose_t* pose_or_null,
                        const double* d_n_close, double d_max, int compute_cov, far_insert_stats_t* d_stats,
                        void* stream);
int far_map_insert_asmd_dev(far_map_t* map, const float* d_xyz, int64_t n, int stride, const far_pose_t* d_pose,
                            const double* d_n_close, double d_max, int compute_cov, far_insert_stats_t* d_stats,
                            void* stream);

/* ---- one frame through the whole path (the LiDAR scan callback) -----------------------------
 * far_frontend_process runs the frame as ONE CUDA GRAPH (cfg.use_graph; captured on the second frame that uses the same
 * scan buffer, stride and result pointer, replayed from then on: per frame a 120-byte parameter upload and one graph
 * launch) or, equivalently, as a stream of launches.  Either way, in stream order and with NO host synchronisation:
 * far_voxelize (ds_voxel) ->
 * scan-local map of the raw scan + far_map_knn_cov of the downsampled points (Sigma_s) ->
 * far_gicp_register against the frontend's map from init_pose -> (update_map) far_map_insert of the raw scan at
 * the registered pose with covariances (cfg.asmd: far_asmd_density of the scan-local map about the sensor, then
 * far_map_insert_asmd) + far_map_prune about it.  Sizes and the registered pose
 * flow between the stages through device memory.  d_out (device, nullable = internal buffer) receives the
 * registration result.  The _host variant takes a HOST scan (pinned for a truly asynchronous copy) and a HOST
 * result struct: it uploads, runs the chain, downloads the result and synchronises the stream. */
typedef struct {
    far_map_config_t map;       /* the local submap (with_cov is forced to 1)                          */
    float ds_voxel;             /* downsampling voxel of far_voxelize; 0 -> map.voxel_size             */
    int64_t max_scan_points;    /* capacity of the per-frame buffers                                   */
    double prune_radius;        /* <= 0: no pruning                                                    */
    int32_t max_iters;          /* GICP iteration limit (R14)                                          */
    int32_t update_map;         /* 0: register only                                                    */
    far_gicp_options_t gicp;
    int32_t asmd;               /* 1: map update with the Adaptive Submap Density limit (R17) */
    double asmd_r_close;        /* "close range of the current scan" [m] for the density; 0 -> 10         */
    double asmd_d_max;          /* range at which the linear decay reaches the lower bound; 0 -> 100       */
    int32_t use_graph;          /* 1: the frame is captured as ONE CUDA graph and replayed; 0: stream of launches */
} far_frontend_config_t;
typedef struct far_frontend far_frontend_t;
int far_frontend_create(far_frontend_t** out, const far_frontend_config_t* cfg);
int far_frontend_destroy(far_frontend_t* f);
far_map_t* far_frontend_map(far_frontend_t* f);   /* borrowed handle, e.g. to preload the map with far_map_insert */
/* 1: frames are being replayed from the captured CUDA graph; 0: no graph yet (it is captured when a frame repeats the
 * previous frame's scan buffer, stride and result pointer); -1: the runtime refused the capture, frames run as a stream of
 * launches */
int far_frontend_graph_state(const far_frontend_t* f);
/* Statistics of the last frame's map update (accepted, new voxels, dropped because full, invalid) copied to HOST memory;
 * synchronises the stream (a diagnostic read, not part of the frame).  A full submap is also reported as FAR_ERR_FULL
 * (see the enum): exactly by far_frontend_process_host (it synchronises), from the mirrored flag by far_frontend_process */
int far_frontend_insert_stats(far_frontend_t* f, far_insert_stats_t* h_out, void* stream);
int far_frontend_process(far_frontend_t* f, const float* d_scan, int64_t n, int stride, const far_pose_t* init_pose,
                         double sigma, far_gicp_result_t* d_out, void* stream);
int far_frontend_process_host(far_frontend_t* f, const float* h_scan, int64_t n, int stride,
                              const far_pose_t* init_pose, double sigma, far_gicp_result_t* h_out, void* stream);
/* the whole LiDAR scan callback of PAPER.md:54-109 including its first step: far_undistort of the raw sweep
 * (d_time, dt_ref, motion as in far_undistort) into an internal buffer, then far_frontend_process on the result */
int far_frontend_process_sweep(far_frontend_t* f, const float* d_scan, const float* d_time, int64_t n, int stride,
                               double dt_ref, const far_motion_t* motion, const far_pose_t* init_pose, double sigma,
                               far_gicp_result_t* d_out, void* stream);

/* Adaptive threshold of Vizzo et al. [1] as read in R10.  HOST-only FP64 helper (20 lines of
 * boundary logic, not a kernel): sigma = sqrt(mean delta_i^2) over recorded deviations delta_i > min_motion,
 * delta = |dt| + 2 max_range sin(theta/2) of pred^-1 * registered; sigma0 until one is recorded. */
far_threshold_t* far_threshold_create(double sigma0, double min_motion, double max_range);
void far_threshold_destroy(far_threshold_t*);
void far_threshold_update(far_threshold_t*, const far_pose_t* predicted, const far_pose_t* registered);
double far_threshold_sigma(const far_threshold_t*);

/* ---- Sensor Fusion backend (Eq. 7-11; R18-R20).  HOST-only FP64 module, outside the
 * GPU hot path ("a small host-side module"): kinematic EKF at a fixed rate with the IMU as control input, corrected by the
 * registered LiDAR pose and velocity with delay compensation and measurement up-sampling.  It supplies what the hot
 * path consumes: the initial guess T_t of the registration and the velocity history of the undistortion.
 *   state x = (t, theta, v): position (map), Euler angles (roll, pitch, yaw; R = Rz Ry Rx), velocity (body)   Eq. 8
 *   predict: x += dt [R(theta) v ; E(theta)(w_m - w_b) ; -[w_m]x v + (a_m - a_b) + g(theta)]                  Eq. 9 (R18)
 *   measurement z = (t_L, theta_L, [theta_ref], v_L), h = row selection                                     Eq. 10 (R19)
 *   delayed measurement taken at cycle s: z_k = z_s + h(x_k|k-1) - h(x_s); applied over n_up cycles with
 *   covariance n_up R (R20)                                                                                  Eq. 11
 * theta_ref (reference roll/pitch of [31],[32]) is an optional INPUT: its formulas are not in the paper. */
typedef struct far_ekf far_ekf_t;
far_ekf_t* far_ekf_create(const double x0[9], const double P0_diag[9], const double Q_diag[9], double dt, int32_t n_up,
                          const double accel_bias_or_null[3], const double gyro_bias_or_null[3]);
void far_ekf_destroy(far_ekf_t*);
/* one cycle: prediction with the IMU sample, then the pending (up-sampled) corrections.  Returns the new cycle index. */
int64_t far_ekf_predict(far_ekf_t*, const double accel_m[3], const double gyro_m[3]);
/* queue a LiDAR measurement taken at cycle `cycle_s` (0 <= current - cycle_s < 512): pose T_L, velocity v_L (Eq. 7),
 * optional reference (roll, pitch), variances in the order of z (9 values, or 11 with theta_ref).  FAR_ERR_ARG if the
 * cycle is no longer in the state history. */
int far_ekf_push_lidar(far_ekf_t*, const far_pose_t* T_L, const double v_L[3], const double theta_ref_or_null[2],
                       const double R_diag[], int64_t cycle_s);
/* current estimate: x[9], P[81] row-major (nullable), cycle index (nullable) */
int far_ekf_state(const far_ekf_t*, double x[9], double* P_or_null, int64_t* cycle_or_null);
/* the state as a pose (R(theta), t): the initial guess T_t of far_gicp_register */
int far_ekf_pose(const far_ekf_t*, far_pose_t* out);
/* the last m cycles as (time = cycle * dt, body twist (v, w_m - w_b)) for far_motion_fit ("velocity history
 * of the Sensor Fusion"); returns the number of samples written (<= m) */
int far_ekf_velocity_history(const far_ekf_t*, int32_t m, double* times, double* vel6);
/* Eq. 7: v_L = R_L,t^-1 (t_t - t_{t-1}) / dt */
int far_lidar_velocity(const far_pose_t* T_t, const far_pose_t* T_prev, double dt, double v_out[3]);
/* exposed for tests: Eq. 9 and its analytic Jacobian F (row-major 9x9) at (x, u = (a_m, w_m)) with zero biases */
int far_ekf_model(const double x[9], const double u[6], double dt, double x_next[9], double F[81]);

#ifdef __cplusplus
}
#endif
#endif
