// far_internal.h -- host-side handle of a map and helpers shared by the translation units of libfar.so.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "far_common.cuh"

struct far_map {
    far_map_config_t cfg;
    far::MapView view;          // device pointers + constants, passed by value to kernels
    uint32_t* d_touched;        // [max_batch] slots that received their first new point in the chunk
    uint32_t* d_cov_list;       // [max_batch] uint4 covariance tasks {key, bucket, c0 | n_new << 8}: the voxels an insert added points to
    uint32_t *d_sp_cnt, *d_sp_vt, *d_sp_ptb, *d_sp_start, *d_sp_seg;   // scratch of the regular-spacing insert (min_spacing > 0)
    void* d_gicp_partials;      // tagged reduction rows + published pose of the cooperative GICP kernel (far_gicp.cu)
    int gicp_max_grid;          // co-resident blocks of the GICP kernel on this device
    int64_t max_batch;
    far::Mailbox* h_mail;       // pinned, mapped host memory the device reports into (full flag, renumbered id counter)
    uint64_t next_id_ub;        // host-side UPPER BOUND of the device-resident id counter (exact unless a renumber is in flight)
    uint64_t offered_total;     // points offered since create / clear
    uint64_t offered_at_renumber;   // value of offered_total when the last renumber pass was enqueued
    uint64_t renumber_every;    // a renumber pass is enqueued before the insert that would exceed this many offered points
    uint32_t renumber_seen;     // mailbox sequence word (2 x passes completed) already looked at
    uint32_t renumber_enqueued; // renumber passes enqueued on this map since create
    uint32_t renumber_ignore;   // passes up to this ordinal were enqueued before the last snapshot restore: never folded
    int device;
    int sm_count;
    int l2_bytes;               // size of the device's L2 (chooses the occupancy-bitmap path of far_map_nn)
};

namespace far {

void set_cuda_error(cudaError_t e, const char* where);

#define FAR_CUDA(call)                                   \
    do {                                                 \
        cudaError_t e_ = (call);                         \
        if (e_ != cudaSuccess) {                         \
            far::set_cuda_error(e_, #call);              \
            return FAR_ERR_CUDA;                         \
        }                                                \
    } while (0)

// Launch accounting (always on: one relaxed counter) and optional per-kernel timing with CUDA events recorded on
// the launching stream (far_profile_enable / far_profile_collect): the tracing facility bench.py reads the
// per-kernel durations from.  Disabled, a LaunchScope costs one atomic increment.
struct LaunchScope {
    LaunchScope(const char* name, cudaStream_t st);
    ~LaunchScope();
    int rec_;
    cudaStream_t st_;
};

#define FAR_LAUNCH(kernel, grid, block, smem, st, ...)        \
    do {                                                      \
        far::LaunchScope ls_(#kernel, st);                    \
        kernel<<<grid, block, smem, st>>>(__VA_ARGS__);       \
    } while (0)

inline int grid_for(int64_t n, int block) { return (int)((n + block - 1) / block); }

// launch helpers implemented in far_query.cu (used by far_map.cu for the covariances of accepted points)
int launch_knn_cov_refs(const far_map* map, const uint32_t* d_refs, const unsigned int* d_n, int64_t n_max,
                        cudaStream_t stream);
int launch_knn_cov_new_ids(const far_map* map, cudaStream_t stream);
// implemented in far_gicp.cu: sizes the cooperative grid, allocates the reduction scratch of a map
int gicp_setup(far_map* map);

// internal forms of the public calls with the point count (and sigma) read from DEVICE memory in stream order: what the
// frame graph of far_frontend.cu replays.  n is then the capacity the launch is sized for, the work is min(n, *d_n)
int voxelize_impl(const float* d_xyz, int64_t n, const int64_t* d_n, int stride, float voxel, float* d_out_xyz, int32_t* d_out_index,
                  int64_t* d_n_out, void* d_workspace, size_t* workspace_bytes, void* stream);
int insert_impl(far_map* m, const float* d_xyz, int64_t n, const int64_t* d_n, int stride, int pose_mode, const far_pose_t* hpose,
                const far_pose_t* d_pose, int compute_cov, far_insert_stats_t* d_stats, void* stream, const double* d_n_close,
                double d_max);
int gicp_launch(const far_map* map, const float* d_scan, const float* d_cov6, const uint8_t* d_valid, int64_t n, const int64_t* d_n,
                int stride, const far_pose_t* hpose, const far_pose_t* d_pose, double sigma, const double* d_sigma, int max_iters,
                int linearize_only, const far_gicp_options_t* opts, far_gicp_result_t* d_out, void* stream);
// kernels launched through FAR_LAUNCH so far (also counts what a replayed frame graph launches)
long long launch_counter();
void launch_counter_add(long long n);
bool profiling_enabled();

}  // namespace far
