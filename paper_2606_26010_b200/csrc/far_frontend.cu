// far_frontend.cu -- one LiDAR frame through the whole hot path as ONE CUDA GRAPH (host code only: it strings the
// kernels of the other translation units together, nothing is computed here).
//
// PAPER.md:54-109 (LiDAR scan callback): [downsample, :171] -> Cov-Calc on a scan-local cuVoxelMap (:76) ->
// GICP against the local submap from the predicted pose (:76-100) -> submap update at the registered pose:
// capped insert, covariances of the added points, range pruning (:109).  Every stage reads its sizes, the predicted pose,
// sigma and the registered pose from device memory, so the chain needs no host synchronisation between stages and --
// is captured once and replayed: per frame the host uploads a 120-byte parameter block and issues one
// cudaGraphLaunch (about 20 runtime calls otherwise, more host time than the device needs for the frame).  The graph is
// keyed by the scan buffer, stride and result pointer and re-captured when they change; launches are sized for
// max_scan_points and clamp to the frame's point count on the device.
#include <cstring>
#include <new>

#include "far_internal.h"

// what changes from frame to frame, in device memory
struct FrameParams {
    int64_t n;               // points in the scan
    far_pose_t init;         // predicted pose (the EKF prior)
    double sigma;            // adaptive threshold
};

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
    cudaStream_t side2;      // third: takes that role while `side` captures the frame graph
    cudaEvent_t ev_fork, ev_join, ev_fork2, ev_join2;
    double* d_asmd;          // [2] n_close, number of close voxels (far_asmd_density)
    float* d_undist;         // undistorted sweep [max_scan_points * 3] (far_frontend_process_sweep)
    far_insert_stats_t* d_insert_stats;   // statistics of the frame's map update (far_frontend_insert_stats)
    FrameParams* d_fp;
    FrameParams* h_fp;       // pinned staging of the frame parameters and of the result for the _host variant (which
    far_gicp_result_t* h_res; //   synchronises every frame, so one slot each is enough): a pageable source or target makes the copy a slow one
    // the captured frame
    cudaGraph_t graph;
    cudaGraphExec_t gexec;
    const float* g_scan;     // key of the captured graph
    int g_stride;
    far_gicp_result_t* g_out;
    long long g_kernels;     // kernels one replay launches
    int graph_state;         // 0: not captured yet (the next frame with a repeated key captures), 1: usable, -1: capture refused
    const float* last_scan;  // key of the previous frame (a graph is captured when a key repeats)
    int last_stride;
    int local_dirty;         // 1: a frame aborted between the scan-local insert and its clear (the next frame clears first)
    far_gicp_result_t* last_out;
};

extern "C" {

int far_frontend_destroy(far_frontend_t* f) {
    if (!f) return FAR_OK;
    far_map_destroy(f->map);
    far_map_destroy(f->local);
    if (f->gexec) cudaGraphExecDestroy(f->gexec);
    if (f->graph) cudaGraphDestroy(f->graph);
    if (f->ev_fork) cudaEventDestroy(f->ev_fork);
    if (f->ev_join) cudaEventDestroy(f->ev_join);
    if (f->ev_fork2) cudaEventDestroy(f->ev_fork2);
    if (f->ev_join2) cudaEventDestroy(f->ev_join2);
    if (f->side) cudaStreamDestroy(f->side);
    if (f->side2) cudaStreamDestroy(f->side2);
    cudaFree(f->d_ws); cudaFree(f->d_scan); cudaFree(f->d_ds_xyz); cudaFree(f->d_ds_index); cudaFree(f->d_n_ds);
    cudaFree(f->d_cov6); cudaFree(f->d_valid); cudaFree(f->d_result); cudaFree(f->d_asmd); cudaFree(f->d_undist); cudaFree(f->d_insert_stats); cudaFree(f->d_fp);
    if (f->h_fp) cudaFreeHost(f->h_fp);
    if (f->h_res) cudaFreeHost(f->h_res);
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
        lc.min_spacing = 0.0;       // R8/R21: Cov-Calc looks for the k nearest RAW scan points; spacing shapes the submap only
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
    alloc((void**)&f->d_fp, sizeof(FrameParams));
    if (e == cudaSuccess) e = cudaHostAlloc((void**)&f->h_fp, sizeof(FrameParams), cudaHostAllocDefault);
    if (e == cudaSuccess) e = cudaHostAlloc((void**)&f->h_res, sizeof(far_gicp_result_t), cudaHostAllocDefault);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&f->side, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&f->side2, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&f->ev_fork, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&f->ev_join, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&f->ev_fork2, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&f->ev_join2, cudaEventDisableTiming);
    if (rc != FAR_OK || e != cudaSuccess) {
        if (e != cudaSuccess) far::set_cuda_error(e, "cudaMalloc in far_frontend_create");
        far_frontend_destroy(f);
        return rc != FAR_OK ? rc : FAR_ERR_CUDA;
    }
    *out = f;
    return FAR_OK;
}

far_map_t* far_frontend_map(far_frontend_t* f) { return f ? f->map : nullptr; }

int far_frontend_graph_state(const far_frontend_t* f) { return f ? f->graph_state : 0; }

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

}  // extern "C"

// the stages of one frame, enqueued on `st`; n_cap sizes the launches, the work is min(n_cap, d_fp->n)
static int frame_chain(far_frontend* f, const float* d_scan, int64_t n_cap, int stride, far_gicp_result_t* res, cudaStream_t st) {
    void* stream = (void*)st;
    const int64_t* d_n = &f->d_fp->n;
    bool full = false;
    // A1/A2 downsampling and the scan-local map are independent until Cov-Calc needs both: fork the downsampling onto
    // the side stream, build the local map on the caller's stream, join before far_map_knn_cov (still no host sync)
    FAR_CUDA(cudaEventRecord(f->ev_fork, st));
    FAR_CUDA(cudaStreamWaitEvent(f->side, f->ev_fork, 0));
    size_t ws = f->ws_bytes;
    FAR_STAGE(far::voxelize_impl(d_scan, n_cap, d_n, stride, f->cfg.ds_voxel, f->d_ds_xyz, f->d_ds_index, f->d_n_ds, f->d_ws, &ws, (void*)f->side));
    FAR_CUDA(cudaEventRecord(f->ev_join, f->side));
    // A7: Sigma_s from a scan-local map of the raw scan.  The scan-local map is EMPTY here: it is created
    // empty and every frame clears it again once it has been used (below, beside the submap update)
    if (f->local_dirty) FAR_STAGE(far_map_clear(f->local, stream));
    f->local_dirty = 1;
    FAR_STAGE(far::insert_impl(f->local, d_scan, n_cap, d_n, stride, 0, nullptr, nullptr, 0, nullptr, stream, nullptr, 1.0));
    FAR_CUDA(cudaStreamWaitEvent(st, f->ev_join, 0));
    if (n_cap > 0) FAR_STAGE(far_map_knn_cov_dev(f->local, f->d_ds_xyz, f->d_n_ds, n_cap, 3, f->d_cov6, f->d_valid, stream));
    // A6, A8-A10: registration from the predicted pose
    FAR_STAGE(far::gicp_launch(f->map, f->d_ds_xyz, f->d_cov6, f->d_valid, n_cap, f->d_n_ds, 3, nullptr, &f->d_fp->init, 0.0, &f->d_fp->sigma,
                               f->cfg.max_iters, 0, &f->cfg.gicp, res, stream));
    const double* d_n_close = nullptr;
    if (f->cfg.update_map && f->cfg.asmd) {
        // density "in a close range of the current scan" = scan-local map about the sensor origin
        const double origin[3] = {0.0, 0.0, 0.0};
        FAR_STAGE(far_asmd_density(f->local, origin, f->cfg.asmd_r_close, f->d_asmd, stream));
        d_n_close = f->d_asmd;
    }
    // the scan-local map has served: it is emptied for the next frame on the side stream, beside the submap update (off
    // the critical path; forked AFTER the registration so that it never delays the cooperative launch)
    FAR_CUDA(cudaEventRecord(f->ev_fork2, st));
    FAR_CUDA(cudaStreamWaitEvent(f->side, f->ev_fork2, 0));
    FAR_STAGE(far_map_clear(f->local, (void*)f->side));
    FAR_CUDA(cudaEventRecord(f->ev_join2, f->side));
    f->local_dirty = 0;
    // A3-A5, A7: submap update at the registered pose
    if (f->cfg.update_map) {
        FAR_STAGE(far::insert_impl(f->map, d_scan, n_cap, d_n, stride, 2, nullptr, &res->pose, 1, f->d_insert_stats, stream, d_n_close,
                                   f->cfg.asmd_d_max));
        if (f->cfg.prune_radius > 0.0) FAR_STAGE(far_map_prune_dev(f->map, &res->pose, f->cfg.prune_radius, nullptr, stream));
    }
    FAR_CUDA(cudaStreamWaitEvent(st, f->ev_join2, 0));
    return full ? FAR_ERR_FULL : FAR_OK;
}

extern "C" {

}  // extern "C"

// pinned_params: the caller synchronises before the next frame, so the parameters may go through the frontend's one
// pinned slot (a truly asynchronous copy); otherwise they are staged by the runtime from the stack before the call returns
static int frontend_process_impl(far_frontend_t* f, const float* d_scan, int64_t n, int stride, const far_pose_t* init_pose,
                                 double sigma, far_gicp_result_t* d_out, void* stream, bool pinned_params) {
    if (!f || !init_pose || n < 0 || n > f->cfg.max_scan_points || (n > 0 && !d_scan) || (stride != 3 && stride != 4) || !(sigma > 0.0))
        return FAR_ERR_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    // an empty frame may come without a scan pointer.  Every stage is sized for max_scan_points and reads the real count
    // (0) on the device, so the launches still want a valid address: the frontend's own staging buffer stands in (it holds
    // max_scan_points x 4 floats, enough for either stride, and is never read when the count is 0)
    if (!d_scan) d_scan = f->d_scan;
    far_gicp_result_t* res = d_out ? d_out : f->d_result;
    FrameParams hp;
    FrameParams* src = pinned_params ? f->h_fp : &hp;
    src->n = n; src->init = *init_pose; src->sigma = sigma;
    FAR_CUDA(cudaMemcpyAsync(f->d_fp, src, sizeof(hp), cudaMemcpyHostToDevice, st));
    const int64_t n_cap = f->cfg.max_scan_points;
    far_map_t* M = f->map;
    // replay is possible when nothing the host decides per frame is due: id renumbering (R22) and the id-range check
    const bool id_ok = !f->cfg.update_map || (M->next_id_ub + (uint64_t)n_cap <= 0xFFFFFFFFull &&
                                              M->offered_total - M->offered_at_renumber + (uint64_t)n_cap <= M->renumber_every);
    const bool same_key = f->last_scan == d_scan && f->last_stride == stride && f->last_out == res;
    f->last_scan = d_scan; f->last_stride = stride; f->last_out = res;
    if (f->cfg.use_graph && id_ok && !far::profiling_enabled() && f->graph_state >= 0) {
        if (f->graph_state == 1 && !(f->g_scan == d_scan && f->g_stride == stride && f->g_out == res)) {
            cudaGraphExecDestroy(f->gexec); cudaGraphDestroy(f->graph);
            f->gexec = nullptr; f->graph = nullptr; f->graph_state = 0;
        }
        if (f->graph_state == 0 && same_key) {
            // second frame on the same buffers: capture it (the first ran directly and did every one-time initialisation)
            const long long k0 = far::launch_counter();
            const uint64_t ub = M->next_id_ub, off = M->offered_total;       // the capture's bookkeeping is redone per replay
            // captured on a stream of the frontend's own (the caller's may be the legacy default stream, which cannot
            // capture); the graph is launched into the caller's stream
            cudaError_t e = cudaStreamBeginCapture(f->side, cudaStreamCaptureModeThreadLocal);
            int rc = FAR_ERR_CUDA;
            if (e == cudaSuccess) {
                cudaStream_t s2 = f->side;
                f->side = f->side2;                                    // the chain forks onto the other internal stream
                rc = frame_chain(f, d_scan, n_cap, stride, res, s2);
                f->side = s2;
                e = cudaStreamEndCapture(f->side, &f->graph);
            }
            if (e != cudaSuccess) far::set_cuda_error(e, "capturing the frame graph");
            M->next_id_ub = ub; M->offered_total = off;
            f->g_kernels = far::launch_counter() - k0;
            far::launch_counter_add(-f->g_kernels);
            if (e == cudaSuccess && (rc == FAR_OK || rc == FAR_ERR_FULL) && f->graph) e = cudaGraphInstantiate(&f->gexec, f->graph, 0);
            if (e == cudaSuccess && (rc == FAR_OK || rc == FAR_ERR_FULL) && f->gexec) {
                f->graph_state = 1; f->g_scan = d_scan; f->g_stride = stride; f->g_out = res;
            } else {
                if (f->graph) { cudaGraphDestroy(f->graph); f->graph = nullptr; }
                f->gexec = nullptr;
                // the runtime refused the capture: stay on the stream path for good.  A stage that rejected its ARGUMENTS
                // says nothing about capturing: this frame runs (and fails) on the stream path, a later one may capture
                f->graph_state = (e == cudaSuccess && rc == FAR_ERR_ARG) ? 0 : -1;
                cudaGetLastError();
            }
        }
        if (f->graph_state == 1) {
            FAR_CUDA(cudaGraphLaunch(f->gexec, st));
            far::launch_counter_add(f->g_kernels);
            if (f->cfg.update_map) { M->next_id_ub += (uint64_t)n_cap; M->offered_total += (uint64_t)n_cap; }
            f->local->next_id_ub = 0; f->local->offered_total = 0; f->local->offered_at_renumber = 0;     // inserted, then cleared
            return far_map_status(M);
        }
    }
    return frame_chain(f, d_scan, n_cap, stride, res, st);
}

extern "C" {

int far_frontend_process(far_frontend_t* f, const float* d_scan, int64_t n, int stride, const far_pose_t* init_pose,
                         double sigma, far_gicp_result_t* d_out, void* stream) {
    return frontend_process_impl(f, d_scan, n, stride, init_pose, sigma, d_out, stream, false);
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
    const int rc = frontend_process_impl(f, f->d_scan, n, stride, init_pose, sigma, f->d_result, stream, true);
    if (rc != FAR_OK && rc != FAR_ERR_FULL) return rc;
    FAR_CUDA(cudaMemcpyAsync(f->h_res, f->d_result, sizeof(far_gicp_result_t), cudaMemcpyDeviceToHost, st));
    FAR_CUDA(cudaStreamSynchronize(st));
    memcpy(h_out, f->h_res, sizeof(far_gicp_result_t));
    return far_map_status(f->map);      // after the sync the mirrored flag is this frame's: FAR_ERR_FULL if it dropped points
}

}  // extern "C"
