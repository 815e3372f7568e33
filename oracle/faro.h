/*
 * faro.h -- C ABI of the ORACLE (test infrastructure, NOT the product).
 *
 * A plain, slow, single-source FP64 CPU restatement of the FAR-LIO front-end hot
 * path, written from the paper text (/root/reference/PAPER.md, cited below as
 * PAPER.md:<line>) and the readings recorded in DESIGN.md.  It shares no code,
 * header, table or helper with the CUDA path in paper_2606_26010_b200/ and must
 * only ever be called from tests/, __graft_entry__.smoke() and the cpu_baseline /
 * --impl reference legs of bench.py.
 *
 * All pointers are HOST pointers.  Points are fp32, `stride` floats apart (3 or 4).
 * Poses are map_from_sensor, R row-major.  Every function returns 0 on success.
 */
#ifndef FARO_H
#define FARO_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct { double R[9]; double t[3]; } faro_pose_t;

typedef struct {
    int64_t n_offered, n_accepted, n_new_voxels, n_dropped_full, n_invalid;
} faro_insert_stats_t;

typedef struct {
    int64_t n_voxels_removed, n_points_removed, n_voxels_left, n_points_left;
} faro_prune_stats_t;

enum { FARO_KERNEL_CAUCHY = 0, FARO_KERNEL_GEMAN_MCCLURE = 1, FARO_KERNEL_NONE = 2 };
enum { FARO_OK = 0, FARO_ERR_ARG = 1, FARO_ERR_RANGE = 4, FARO_ERR_DEGENERATE = 5 };

typedef struct {
    int32_t kernel;      /* FARO_KERNEL_* ; PAPER.md:88-90 (Eq. 5) Cauchy is the paper's */
    double conv_eps;     /* 5e-3 */
    double tau_mult;     /* gate tau = tau_mult * sigma (reading A-6: 3) */
    double kappa_div;    /* kernel scale kappa = sigma / kappa_div (reading A-6: 3) */
} faro_gicp_options_t;

typedef struct {
    faro_pose_t pose;
    double H[36];
    double b[6];
    double chi2;
    int32_t n_inliers, iters, converged, status;
} faro_gicp_result_t;

typedef struct faro_map faro_map_t;
typedef struct faro_threshold faro_threshold_t;

/* A1  PAPER.md:62 "custom key, defined by the 3D indices of a voxel" */
int faro_keys(const float* xyz, int64_t n, int stride, float voxel, uint64_t* keys, uint8_t* valid);
uint64_t faro_pack_key(int32_t kx, int32_t ky, int32_t kz);
void faro_unpack_key(uint64_t key, int32_t* k3);

/* A2  PAPER.md:171 (downsampling); reading: first point per voxel, ascending source index */
int faro_voxelize(const float* xyz, int64_t n, int stride, float voxel,
                  float* out_xyz /* n*3 */, int32_t* out_index /* n */, int64_t* n_out);

/* A3/A4/A5 */
faro_map_t* faro_map_create(float voxel, int32_t cap, int32_t k_cov, double cov_eps);
void faro_map_destroy(faro_map_t*);
/* deep copy of a map (contents, covariances, id counter, configuration); NULL in -> NULL out.  Bookkeeping only. */
faro_map_t* faro_map_clone(const faro_map_t*);
/* R21: s > 0: an offered point is stored only if no point already stored in its own voxel is closer than s
 * (FP64 squared distance as R6, strict <), tested in index order after the cap; s = 0 (default): the plain capped insert */
void faro_map_set_min_spacing(faro_map_t*, double s);
int faro_map_insert(faro_map_t*, const float* xyz, int64_t n, int stride, const faro_pose_t* pose_or_null,
                    int compute_cov, faro_insert_stats_t* stats);
int faro_map_prune(faro_map_t*, const double center[3], double radius, faro_prune_stats_t* stats);
int faro_map_size(const faro_map_t*, int64_t* n_voxels, int64_t* n_points, uint64_t* next_id);
/* R22: subtract the smallest stored id from every stored id and from the id counter (empty map: counter -> 0) */
int faro_map_renumber(faro_map_t*, uint64_t* subtracted);
/* export sorted by key; points: n_voxels*cap*4 floats (x,y,z,id bits), unused entries zero/0xFFFFFFFF */
int faro_map_export(const faro_map_t*, uint64_t* keys, int32_t* counts, float* points4,
                    float* cov6 /* nullable, n_voxels*cap*6 */, uint8_t* cov_valid /* nullable */);

/* A6  PAPER.md:62,80 : 27-voxel nearest neighbour, (d2,id) lexicographic */
int faro_map_nn(const faro_map_t*, const float* q, int64_t m, int stride, uint32_t* id, float* d2, int nthreads);
/* pin helper: brute force over ALL stored points with the key-adjacency filter */
int faro_map_nn_brute(const faro_map_t*, const float* q, int64_t m, int stride, uint32_t* id, float* d2);
/* pin helper: the k nearest ids (0xFFFFFFFF padded) and FP64 squared distances */
int faro_map_knn(const faro_map_t*, const float* q, int64_t m, int stride, int32_t k, uint32_t* ids, double* d2);

/* A7  PAPER.md:68-76 (Eq. 1) */
int faro_map_knn_cov(const faro_map_t*, const float* q, int64_t m, int stride, float* cov6, uint8_t* valid, int nthreads);
/* pin helper: Eq. 1 on an explicit k x 3 neighbour list (FP64 out) */
int faro_cov_from_points(const float* pts, int32_t k, int stride, double eps, double* cov6_out);

/* A8-A10  PAPER.md:76-100 (Eq. 2-6) */
int faro_gicp_linearize(const faro_map_t*, const float* scan, const float* scan_cov6, const uint8_t* scan_valid,
                        int64_t n, int stride, const faro_pose_t* pose, double sigma,
                        const faro_gicp_options_t* opts, faro_gicp_result_t* out, int nthreads);
int faro_gicp_register(const faro_map_t*, const float* scan, const float* scan_cov6, const uint8_t* scan_valid,
                       int64_t n, int stride, const faro_pose_t* init_pose, double sigma, int max_iters,
                       const faro_gicp_options_t* opts, faro_gicp_result_t* out, int nthreads);
void faro_gicp_default_options(faro_gicp_options_t*);
/* pin helpers */
void faro_se3_exp(const double delta[6], faro_pose_t* out);
double faro_robust_weight(int kernel, double e2, double kappa);
/* per-correspondence data of one linearisation, for finite-difference pins:
   for each source point: used flag, p (transformed fp32 widened), r, M(9), w */
int faro_gicp_correspondences(const faro_map_t*, const float* scan, const float* scan_cov6, const uint8_t* scan_valid,
                              int64_t n, int stride, const faro_pose_t* pose, double sigma,
                              const faro_gicp_options_t* opts, uint8_t* used, double* p3, double* r3,
                              double* M9, double* w, uint32_t* id);

/* adaptive threshold of Vizzo et al. [1] as read in DESIGN.md */
faro_threshold_t* faro_threshold_create(double sigma0, double min_motion, double max_range);
void faro_threshold_destroy(faro_threshold_t*);
void faro_threshold_update(faro_threshold_t*, const faro_pose_t* predicted, const faro_pose_t* registered);
double faro_threshold_sigma(const faro_threshold_t*);

/* ---- SURVEY 8(f)-2  PAPER.md:56 (Preprocessing & Undistortion); readings R15/R16 in DESIGN.md --------------
 * "We perform a linear regression on both the linear and angular velocities ... This continuous motion model is
 * evaluated ... each raw point is undistorted and projected to the frame reference timestamp, which is equal to
 * the scan's final point-timestamp."
 * motion: body twist xi(t) = a + b (t - t_ref), 6-vectors (linear velocity first, then angular velocity). */
typedef struct { double a[6]; double b[6]; } faro_motion_t;
/* R15: ordinary least-squares line per component over m history samples (times[j], vel[j*6 .. j*6+5]);
 * fewer than 2 distinct times -> b = 0, a = mean. */
int faro_motion_fit(const double* times, const double* vel6, int32_t m, double t_ref, faro_motion_t* out);
/* R16: point i was measured at t_first + time[i]; Delta_i = dt_ref - (double)time[i] (dt_ref = t_ref - t_first);
 * Omega_i = a Delta_i - b Delta_i^2 / 2 + [a,b] Delta_i^3 / 12 (Magnus expansion to second order, se(3) bracket);
 * out_i = fl32(Exp(-Omega_i) p_i)  (SE(3) exponential of R12, transform of R4).
 * out_xyz: n*3 floats; non-finite points are copied unchanged. */
int faro_undistort(const float* xyz, const float* time, int64_t n, int stride, double dt_ref,
                   const faro_motion_t* motion, float* out_xyz);

/* ---- SURVEY 8(f)-1  PAPER.md:109 (Adaptive Submap Density); reading R17 -------------------------------------
 * "the average amount of points per voxel in a close range of the current scan is computed ... linear decay (with
 * a lower bound defined by the k = 10 points required to compute the covariances) ... integrated into the
 * corresponding voxels ... as long as the number of points inside it is below N_ASMD."
 * density: mean stored points per voxel over the voxels of `local` whose centre is within r_close of `center`
 * (|(k+0.5)v - c|^2 <= r_close^2, FP64 as in R5); *n_close = cap of `local` if there is no such voxel. */
int faro_asmd_density(const faro_map_t* local, const double center[3], double r_close, double* n_close,
                      int64_t* n_voxels_close);
/* N_ASMD of the voxel with index k3 seen from `center`: clamp(floor(n_close (1 - d/d_max) + 0.5), k_min, cap),
 * d = |(k+0.5)v - center| ; every operation one rounded binary64 operation. */
int32_t faro_asmd_cap(const int32_t k3[3], float voxel, const double center[3], double n_close, double d_max,
                      int32_t k_min, int32_t cap);
/* faro_map_insert with the per-voxel limit N_ASMD (centre = pose->t, or the origin without a pose; k_min = k_cov) */
int faro_map_insert_asmd(faro_map_t*, const float* xyz, int64_t n, int stride, const faro_pose_t* pose_or_null,
                         double n_close, double d_max, int compute_cov, faro_insert_stats_t* stats);

#ifdef __cplusplus
}
#endif
#endif
