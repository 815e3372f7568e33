// far_frontend.cu -- one LiDAR frame through the whole hot path as a single stream-ordered chain (host code
// only: it strings the kernels of the other translation units together, nothing is computed here).
//
// PAPER.md:54-109 (LiDAR scan callback): [downsample, :171] -> Cov-Calc on a scan-local cuVoxelMap (:76) ->
// GICP against the local submap from the predicted pose (:76-100) -> submap update at the registered pose:
// capped insert, covariances of the added points, range pruning (:109).  Every stage reads its sizes and the
// registered pose from device memory, so the chain needs no host synchronisation between stages.
#include <cstring>
#include <new>

#include "far_internal.h"

struct far_frontend {
    far_frontend_config_t cfg;
    far_map_t* map;          // the local submap Q
    far_map_t* local;        // scan-local map used for Sigma_s
    void* d_ws;              // far_voxelize workspace
    size_t ws_bytes;
    float* d_scan;           // staging for host scans [max_scan_points * 4]
    float* d_ds_xyz;         // downsampled scan
    int32_t* d_ds_index;
    int64_t* d_n_ds;
    float* d_cov6;
    uint8_t* d_valid;
    far_gicp_result_t* d_result;
    cudaStream_t side;       // second stream: the downsampling branch runs beside the scan-local map build
    cudaEvent_t ev_fork, ev_join;
    double* d_asmd;          // [2] n_close, number of close voxels (far_asmd_density)
    float* d_undist;         // undistorted sweep [max_scan_points * 3] (far_frontend_process_sweep)
    far_insert_stats_t* d_insert_stats;   // statistics of the frame's map update (far_frontend_insert_stats)
};

extern "C" {

int far_frontend_destroy(far_frontend_t* f) {
    if (!f) return FAR_OK;
    far_map_destroy(f->map);
    far_map_destroy(f->local);
    if (f->ev_fork) cudaEventDestroy(f->ev_fork);
    if (f->ev_join) cudaEventDestroy(f->ev_join);
    if (f->side) cudaStreamDestroy(f->side);
    cudaFree(f->d_ws); cudaFree(f->d_scan); cudaFree(f->d_ds_xyz); cudaFree(f->d_ds_index); cudaFree(f->d_n_ds);
    cudaFree(f->d_cov6); cudaFree(f->d_valid); cudaFree(f->d_result); cudaFree(f->d_asmd); cudaFree(f->d_undist); cudaFree(f->d_insert_stats);
    delete f;
    return FAR_OK;
}

int far_frontend_create(far_frontend_t** out, const far_frontend_config_t* cfg) {
    if (!out || !cfg || cfg->max_scan_points < 1 || cfg->max_iters < 1) return FAR_ERR_ARG;
    *out = nullptr;
    far_frontend* f = new (std::nothrow) far_frontend();
    if (!f) return FAR_ERR_ARG;
    memset(f, 0, sizeof(*f));
    f->cfg = *cfg;
    if (!(f->cfg.ds_voxel > 0.f)) f->cfg.ds_voxel = cfg->map.voxel_size;
    if (!(f->cfg.asmd_r_close > 0.0)) f->cfg.asmd_r_close = 10.0;
    if (!(f->cfg.asmd_d_max > 0.0)) f->cfg.asmd_d_max = 100.0;
    far_map_config_t mc = cfg->map;
    mc.with_cov = 1;
    if (mc.max_batch < cfg->max_scan_points) mc.max_batch = cfg->max_scan_points;
    int rc = far_map_create(&f->map, &mc);
    if (rc == FAR_OK) {
        far_map_config_t lc = cfg->map;
        lc.with_cov = 0;
        lc.max_voxels = cfg->max_scan_points;
        lc.max_load = 0.5f;
        lc.max_batch = cfg->max_scan_points;
        rc = far_map_create(&f->local, &lc);
    }
    if (rc != FAR_OK) { far_frontend_destroy(f); return rc; }
    const int64_t n = cfg->max_scan_points;
    rc = far_voxelize(nullptr, n, 3, f->cfg.ds_voxel, nullptr, nullptr, nullptr, nullptr, &f->ws_bytes, nullptr);
    cudaError_t e = cudaSuccess;
    auto alloc = [&](void** p, size_t bytes) { if (e == cudaSuccess) e = cudaMalloc(p, bytes); };
    alloc(&f->d_ws, f->ws_bytes);
    alloc((void**)&f->d_scan, (size_t)n * 4 * sizeof(float));
    alloc((void**)&f->d_ds_xyz, (size_t)n * 3 * sizeof(float));
    alloc((void**)&f->d_ds_index, (size_t)n * sizeof(int32_t));
    alloc((void**)&f->d_n_ds, sizeof(int64_t));
    alloc((void**)&f->d_cov6, (size_t)n * 6 * sizeof(float));
    alloc((void**)&f->d_valid, (size_t)n);
    alloc((void**)&f->d_result, sizeof(far_gicp_result_t));
    alloc((void**)&f->d_asmd, 2 * sizeof(double));
    alloc((void**)&f->d_undist, (size_t)n * 3 * sizeof(float));
    alloc((void**)&f->d_insert_stats, sizeof(far_insert_stats_t));
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&f->side, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&f->ev_fork, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&f->ev_join, cudaEventDisableTiming);
    if (rc != FAR_OK || e != cudaSuccess) {
        if (e != cudaSuccess) far::set_cuda_error(e, "cudaMalloc in far_frontend_create");
        far_frontend_destroy(f);
        return rc != FAR_OK ? rc : FAR_ERR_CUDA;
    }
    *out = f;
    return FAR_OK;
}

far_map_t* far_frontend_map(far_frontend_t* f) { return f ? f->map : nullptr; }

int far_frontend_insert_stats(far_frontend_t* f, far_insert_stats_t* h_out, void* stream) {
    if (!f || !h_out) return FAR_ERR_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    FAR_CUDA(cudaMemcpyAsync(h_out, f->d_insert_stats, sizeof(*h_out), cudaMemcpyDeviceToHost, st));
    FAR_CUDA(cudaStreamSynchronize(st));
    return FAR_OK;
}

// FAR_ERR_FULL from a stage means "work enqueued, the map has dropped points" (far.h): the chain goes on and the frame
// reports it at the end; every other status aborts the frame
#define FAR_STAGE(call)                                 \
    do {                                                \
        const int rc_ = (call);                         \
        if (rc_ == FAR_ERR_FULL) full = true;           \
        else if (rc_ != FAR_OK) return rc_;             \
    } while (0)

int far_frontend_process(far_frontend_t* f, const float* d_scan, int64_t n, int stride, const far_pose_t* init_pose,
                         double sigma, far_gicp_result_t* d_out, void* stream) {
    if (!f || !init_pose || n < 0 || n > f->cfg.max_scan_points || (n > 0 && !d_scan) || (stride != 3 && stride != 4))
        return FAR_ERR_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    far_gicp_result_t* res = d_out ? d_out : f->d_result;
    bool full = false;
    // A1/A2 downsampling and the scan-local map are independent until Cov-Calc needs both: fork the downsampling onto
    // the side stream, build the local map on the caller's stream, join before far_map_knn_cov (still no host sync)
    FAR_CUDA(cudaEventRecord(f->ev_fork, st));
    FAR_CUDA(cudaStreamWaitEvent(f->side, f->ev_fork, 0));
    size_t ws = f->ws_bytes;
    FAR_STAGE(far_voxelize(d_scan, n, stride, f->cfg.ds_voxel, f->d_ds_xyz, f->d_ds_index, f->d_n_ds, f->d_ws, &ws, (void*)f->side));
    FAR_CUDA(cudaEventRecord(f->ev_join, f->side));
    // A7: Sigma_s from a scan-local map of the raw scan
    FAR_STAGE(far_map_clear(f->local, stream));
    FAR_STAGE(far_map_insert(f->local, d_scan, n, stride, nullptr, 0, nullptr, stream));
    FAR_CUDA(cudaStreamWaitEvent(st, f->ev_join, 0));
    if (n > 0) FAR_STAGE(far_map_knn_cov_dev(f->local, f->d_ds_xyz, f->d_n_ds, n, 3, f->d_cov6, f->d_valid, stream));
    // A6, A8-A10: registration from the predicted pose
    FAR_STAGE(far_gicp_register_dn(f->map, f->d_ds_xyz, f->d_cov6, f->d_valid, f->d_n_ds, n, 3, init_pose, sigma,
                                   f->cfg.max_iters, &f->cfg.gicp, res, stream));
    // A3-A5, A7: submap update at the registered pose
    if (f->cfg.update_map) {
        if (f->cfg.asmd) {
            // density "in a close range of the current scan" = scan-local map about the sensor origin
            const double origin[3] = {0.0, 0.0, 0.0};
            FAR_STAGE(far_asmd_density(f->local, origin, f->cfg.asmd_r_close, f->d_asmd, stream));
            FAR_STAGE(far_map_insert_asmd_dev(f->map, d_scan, n, stride, &res->pose, f->d_asmd, f->cfg.asmd_d_max, 1, f->d_insert_stats, stream));
        } else {
            FAR_STAGE(far_map_insert_dev(f->map, d_scan, n, stride, &res->pose, 1, f->d_insert_stats, stream));
        }
        if (f->cfg.prune_radius > 0.0) FAR_STAGE(far_map_prune_dev(f->map, &res->pose, f->cfg.prune_radius, nullptr, stream));
    }
    return full ? FAR_ERR_FULL : FAR_OK;
}

int far_frontend_process_sweep(far_frontend_t* f, const float* d_scan, const float* d_time, int64_t n, int stride, double dt_ref,
                               const far_motion_t* motion, const far_pose_t* init_pose, double sigma, far_gicp_result_t* d_out,
                               void* stream) {
    if (!f || n < 0 || n > f->cfg.max_scan_points) return FAR_ERR_ARG;
    const int rc = far_undistort(d_scan, d_time, n, stride, dt_ref, motion, f->d_undist, stream);
    if (rc != FAR_OK) return rc;
    return far_frontend_process(f, f->d_undist, n, 3, init_pose, sigma, d_out, stream);
}

int far_frontend_process_host(far_frontend_t* f, const float* h_scan, int64_t n, int stride, const far_pose_t* init_pose,
                              double sigma, far_gicp_result_t* h_out, void* stream) {
    if (!f || !h_out || n < 0 || n > f->cfg.max_scan_points || (n > 0 && !h_scan) || (stride != 3 && stride != 4)) return FAR_ERR_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    if (n > 0) FAR_CUDA(cudaMemcpyAsync(f->d_scan, h_scan, (size_t)n * stride * sizeof(float), cudaMemcpyHostToDevice, st));
    const int rc = far_frontend_process(f, f->d_scan, n, stride, init_pose, sigma, f->d_result, stream);
    if (rc != FAR_OK && rc != FAR_ERR_FULL) return rc;
    FAR_CUDA(cudaMemcpyAsync(h_out, f->d_result, sizeof(far_gicp_result_t), cudaMemcpyDeviceToHost, st));
    FAR_CUDA(cudaStreamSynchronize(st));
    return far_map_status(f->map);      // after the sync the mirrored flag is this frame's: FAR_ERR_FULL if it dropped points
}

}  // extern "C"
