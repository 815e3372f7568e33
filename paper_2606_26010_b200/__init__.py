"""paper_2606_26010_b200 -- thin Python binding of libfar.so (the C ABI declared in include/far.h).

Argument marshalling only: every step of the hot path (voxel keys, hashmap insert/prune, 27-voxel nearest
neighbour, k-NN covariances, GICP linearisation and the Gauss-Newton loop) runs in the hand-written CUDA
kernels of csrc/.  PyTorch supplies device memory and streams; nothing here computes.  There is no CPU
fallback: importing works without a GPU (so the ABI can be inspected), every compute call needs one, and a
missing library raises.

Names follow include/far.h and the paper's notation.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

from . import _build

NO_ID = 0xFFFFFFFF
KERNEL_CAUCHY, KERNEL_GEMAN_MCCLURE, KERNEL_NONE = 0, 1, 2
OK, ERR_ARG, ERR_CUDA, ERR_FULL, ERR_RANGE, ERR_DEGENERATE = 0, 1, 2, 3, 4, 5

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libfar.so")


class Pose(C.Structure):
    _fields_ = [("R", C.c_double * 9), ("t", C.c_double * 3)]

    @staticmethod
    def from_rt(T):
        R, t = T
        p = Pose()
        p.R[:] = np.asarray(R, dtype=np.float64).reshape(9).tolist()
        p.t[:] = np.asarray(t, dtype=np.float64).reshape(3).tolist()
        return p

    def to_rt(self):
        return np.array(self.R[:]).reshape(3, 3), np.array(self.t[:])


class MapConfig(C.Structure):
    _fields_ = [("voxel_size", C.c_float), ("cap", C.c_int32), ("max_voxels", C.c_int64), ("max_load", C.c_float),
                ("with_cov", C.c_int32), ("k_cov", C.c_int32), ("cov_eps", C.c_double), ("max_batch", C.c_int64),
                ("renumber_every", C.c_int64), ("min_spacing", C.c_double)]


class GicpOptions(C.Structure):
    _fields_ = [("kernel", C.c_int32), ("conv_eps", C.c_double), ("tau_mult", C.c_double), ("kappa_div", C.c_double)]


class GicpResult(C.Structure):
    _fields_ = [("pose", Pose), ("H", C.c_double * 36), ("b", C.c_double * 6), ("chi2", C.c_double),
                ("n_inliers", C.c_int32), ("iters", C.c_int32), ("converged", C.c_int32), ("status", C.c_int32)]


class FrontendConfig(C.Structure):
    _fields_ = [("map", MapConfig), ("ds_voxel", C.c_float), ("max_scan_points", C.c_int64), ("prune_radius", C.c_double),
                ("max_iters", C.c_int32), ("update_map", C.c_int32), ("gicp", GicpOptions),
                ("asmd", C.c_int32), ("asmd_r_close", C.c_double), ("asmd_d_max", C.c_double), ("use_graph", C.c_int32)]


class Motion(C.Structure):
    """far_motion_t: body twist xi(t) = a + b (t - t_ref), linear velocity first (R15)"""
    _fields_ = [("a", C.c_double * 6), ("b", C.c_double * 6)]

    @staticmethod
    def from_ab(a, b):
        m = Motion()
        m.a[:] = np.asarray(a, dtype=np.float64).reshape(6).tolist()
        m.b[:] = np.asarray(b, dtype=np.float64).reshape(6).tolist()
        return m

    def to_ab(self):
        return np.array(self.a[:]), np.array(self.b[:])


INSERT_STATS_FIELDS = ("n_offered", "n_accepted", "n_new_voxels", "n_dropped_full", "n_invalid")
PRUNE_STATS_FIELDS = ("n_voxels_removed", "n_points_removed", "n_voxels_left", "n_points_left")
MAP_STATS_FIELDS = ("n_voxels", "n_points", "n_dead_keys", "n_slots", "next_id", "n_keys", "n_free_buckets", "n_fresh_buckets",
                    "n_rehash", "full")
GICP_RESULT_BYTES = C.sizeof(GicpResult)
POSE_BYTES = C.sizeof(Pose)

_lib = None


class FarError(RuntimeError):
    def __init__(self, status, where):
        self.status = status
        msg = lib().far_strerror(status).decode()
        cuda = lib().far_last_cuda_error().decode()
        super().__init__(f"{where}: {msg} (status {status})" + (f" [{cuda}]" if status == ERR_CUDA and cuda else ""))


def lib():
    """Load (building if needed) the in-tree libfar.so.  Raises if it cannot be built or loaded."""
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        vp, i64, i32, f32, f64, ci = C.c_void_p, C.c_int64, C.c_int32, C.c_float, C.c_double, C.c_int
        sig = {
            "far_strerror": (C.c_char_p, [ci]),
            "far_last_cuda_error": (C.c_char_p, []),
            "far_launch_count": (C.c_longlong, []),
            "far_profile_enable": (None, [ci]),
            "far_profile_collect": (ci, [vp, vp, vp, ci]),
            "far_gicp_default_options": (None, [vp]),
            "far_map_create": (ci, [vp, vp]),
            "far_map_destroy": (ci, [vp]),
            "far_map_clear": (ci, [vp, vp]),
            "far_map_insert": (ci, [vp, vp, i64, ci, vp, ci, vp, vp]),
            "far_map_insert_dev": (ci, [vp, vp, i64, ci, vp, ci, vp, vp]),
            "far_map_prune": (ci, [vp, vp, f64, vp, vp]),
            "far_map_prune_dev": (ci, [vp, vp, f64, vp, vp]),
            "far_map_stats": (ci, [vp, vp, vp]),
            "far_map_rehash": (ci, [vp, vp]),
            "far_map_renumber": (ci, [vp, vp]),
            "far_map_status": (ci, [vp]),
            "far_frontend_insert_stats": (ci, [vp, vp, vp]),
            "far_frontend_graph_state": (ci, [vp]),
            "far_map_snapshot_create": (ci, [vp, vp, vp]),
            "far_map_snapshot_restore": (ci, [vp, vp, vp]),
            "far_map_snapshot_destroy": (ci, [vp]),
            "far_map_count27": (ci, [vp, vp, i64, ci, vp, vp, vp]),
            "far_map_export": (ci, [vp, vp, vp, vp, vp, vp, i64, vp, vp]),
            "far_voxel_keys": (ci, [vp, i64, ci, f32, vp, vp]),
            "far_map_nn": (ci, [vp, vp, i64, ci, vp, vp, vp]),
            "far_map_knn_cov": (ci, [vp, vp, i64, ci, vp, vp, vp]),
            "far_map_knn_cov_dev": (ci, [vp, vp, vp, i64, ci, vp, vp, vp]),
            "far_voxelize": (ci, [vp, i64, ci, f32, vp, vp, vp, vp, vp, vp]),
            "far_voxelize_static": (ci, [vp, i64, ci, f32, vp, vp, vp, vp]),
            "far_gicp_linearize": (ci, [vp, vp, vp, vp, i64, ci, vp, f64, vp, vp, vp]),
            "far_gicp_register": (ci, [vp, vp, vp, vp, i64, ci, vp, f64, ci, vp, vp, vp]),
            "far_gicp_register_dev": (ci, [vp, vp, vp, vp, vp, i64, ci, vp, f64, ci, vp, vp, vp]),
            "far_gicp_register_dn": (ci, [vp, vp, vp, vp, vp, i64, ci, vp, f64, ci, vp, vp, vp]),
            "far_frontend_create": (ci, [vp, vp]),
            "far_frontend_destroy": (ci, [vp]),
            "far_frontend_map": (vp, [vp]),
            "far_frontend_process": (ci, [vp, vp, i64, ci, vp, f64, vp, vp]),
            "far_frontend_process_host": (ci, [vp, vp, i64, ci, vp, f64, vp, vp]),
            "far_frontend_process_sweep": (ci, [vp, vp, vp, i64, ci, f64, vp, vp, f64, vp, vp]),
            "far_motion_fit": (ci, [vp, vp, i32, f64, vp]),
            "far_undistort": (ci, [vp, vp, i64, ci, f64, vp, vp, vp]),
            "far_asmd_density": (ci, [vp, vp, f64, vp, vp]),
            "far_map_insert_asmd": (ci, [vp, vp, i64, ci, vp, vp, f64, ci, vp, vp]),
            "far_map_insert_asmd_dev": (ci, [vp, vp, i64, ci, vp, vp, f64, ci, vp, vp]),
            "far_ekf_create": (vp, [vp, vp, vp, f64, i32, vp, vp]),
            "far_ekf_destroy": (None, [vp]),
            "far_ekf_predict": (i64, [vp, vp, vp]),
            "far_ekf_push_lidar": (ci, [vp, vp, vp, vp, vp, i64]),
            "far_ekf_state": (ci, [vp, vp, vp, vp]),
            "far_ekf_pose": (ci, [vp, vp]),
            "far_ekf_velocity_history": (ci, [vp, i32, vp, vp]),
            "far_lidar_velocity": (ci, [vp, vp, f64, vp]),
            "far_ekf_model": (ci, [vp, vp, f64, vp, vp]),
            "far_threshold_create": (vp, [f64, f64, f64]),
            "far_threshold_destroy": (None, [vp]),
            "far_threshold_update": (None, [vp, vp, vp]),
            "far_threshold_sigma": (f64, [vp]),
        }
        for name, (res, args) in sig.items():
            fn = getattr(L, name)
            fn.restype = res
            fn.argtypes = args
        L._far_symbols = tuple(sig)
        _lib = L
    return _lib


def _check(rc, where, full_ok=False):
    """FAR_ERR_FULL from insert / frontend calls means "work enqueued, the map has dropped points" (far.h): those callers
    pass full_ok and get the flag back instead of an exception."""
    if rc == ERR_FULL and full_ok:
        return True
    if rc != OK:
        raise FarError(rc, where)
    return False


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _ptr(t):
    return C.c_void_p(t.data_ptr()) if t is not None else None


def _points(x):
    """Device fp32 (n,3) or (n,4) contiguous tensor -> (tensor, n, stride)."""
    if not isinstance(x, torch.Tensor):
        x = torch.as_tensor(np.ascontiguousarray(x, dtype=np.float32))
    if x.device.type != "cuda":
        x = x.cuda()
    if x.dtype != torch.float32 or not x.is_contiguous():
        x = x.to(torch.float32).contiguous()
    assert x.dim() == 2 and x.shape[1] in (3, 4), tuple(x.shape)
    return x, x.shape[0], x.shape[1]


def _struct_from_tensor(t, cls):
    raw = t.cpu().numpy().tobytes()
    return cls.from_buffer_copy(raw)


def default_options(kernel=KERNEL_CAUCHY, conv_eps=5e-3, tau_mult=3.0, kappa_div=3.0):
    return GicpOptions(kernel, conv_eps, tau_mult, kappa_div)


def result_to_dict(res: GicpResult):
    # one copy of the 456-byte struct: 55 doubles (pose 12, H 36, b 6, chi2) then four int32
    d = np.frombuffer(res, dtype=np.float64, count=55).copy()
    return dict(R=d[0:9].reshape(3, 3), t=d[9:12], H=d[12:48].reshape(6, 6), b=d[48:54], chi2=float(d[54]),
                n_inliers=res.n_inliers, iters=res.iters, converged=res.converged, status=res.status)


def launch_count():
    """far_launch_count: kernels launched by libfar.so in this process so far."""
    return int(lib().far_launch_count())


def profile_enable(on=True):
    lib().far_profile_enable(int(bool(on)))


def profile_collect(max_entries=64):
    """far_profile_collect -> {kernel name: (total_ms, launches)}; synchronises the device."""
    names = (C.c_char_p * max_entries)()
    ms = (C.c_double * max_entries)()
    cnt = (C.c_longlong * max_entries)()
    n = lib().far_profile_collect(names, ms, cnt, max_entries)
    return {names[i].decode(): (ms[i], int(cnt[i])) for i in range(n)}


def voxel_keys(xyz, voxel):
    """far_voxel_keys: packed voxel key per point (uint64 bit pattern in an int64 tensor)."""
    x, n, s = _points(xyz)
    keys = torch.empty(n, dtype=torch.int64, device=x.device)
    _check(lib().far_voxel_keys(_ptr(x), n, s, voxel, _ptr(keys), _stream()), "far_voxel_keys")
    return keys


class Voxelizer:
    """far_voxelize with a reusable workspace sized for up to n_max points."""

    def __init__(self, n_max, device="cuda"):
        self.n_max = int(n_max)
        nbytes = C.c_size_t(0)
        _check(lib().far_voxelize(None, self.n_max, 3, 1.0, None, None, None, None, C.byref(nbytes), None), "far_voxelize(size)")
        self.ws = torch.empty(nbytes.value, dtype=torch.uint8, device=device)
        self.out_xyz = torch.empty((self.n_max, 3), dtype=torch.float32, device=device)
        self.out_index = torch.empty(self.n_max, dtype=torch.int32, device=device)
        self.n_out = torch.zeros(1, dtype=torch.int64, device=device)

    def enqueue(self, xyz, voxel):
        """No host sync: results stay on the device (out_xyz, out_index, n_out)."""
        x, n, s = _points(xyz)
        assert n <= self.n_max
        nbytes = C.c_size_t(self.ws.numel())
        _check(lib().far_voxelize(_ptr(x), n, s, voxel, _ptr(self.out_xyz), _ptr(self.out_index), _ptr(self.n_out),
                                  _ptr(self.ws), C.byref(nbytes), _stream()), "far_voxelize")

    def __call__(self, xyz, voxel):
        self.enqueue(xyz, voxel)
        m = int(self.n_out.item())
        return self.out_xyz[:m].clone(), self.out_index[:m].clone()


def voxelize(xyz, voxel):
    x, n, _ = _points(xyz)
    return Voxelizer(max(n, 1), device=x.device)(x, voxel)


VOXELIZE_STATIC_MAX_POINTS = 262144   # FAR_VOXELIZE_STATIC_MAX_POINTS
VOXELIZE_STATIC_BYTES = 7341568       # FAR_VOXELIZE_STATIC_BYTES: held by every GPU that loads libfar.so


def voxelize_static(xyz, voxel, out_xyz, out_index, n_out):
    """far_voxelize_static: far_voxelize for callers that may not allocate device memory.

    Meant for code that gets its buffers from somewhere else and has no allocator of its own to call: a LiDAR callback
    in a real-time loop (cudaMalloc takes driver locks and may stall the whole device), a plug-in living on its host
    application's GPU memory budget.  The library's own fixed scratch array (about 7 MiB per GPU, shared by all calls)
    replaces the workspace, so the scan is limited to VOXELIZE_STATIC_MAX_POINTS points; more raises FarError(ERR_ARG).
    The caller passes every buffer: `xyz` a CUDA fp32 (n,3|4) tensor, `out_xyz` (>= n,3) fp32, `out_index` (>= n,) int32,
    `n_out` (1,) int64, all on the device; this wrapper creates no tensor and does not synchronise -- results are valid in
    stream order, the count is n_out[0].  Call it once per device at start-up (n = 0 will do): the first call on a device
    looks the scratch address up.  Calls that overlap on one GPU share the scratch and corrupt each other."""
    assert isinstance(xyz, torch.Tensor) and xyz.is_cuda and xyz.dtype == torch.float32 and xyz.is_contiguous()
    assert xyz.dim() == 2 and xyz.shape[1] in (3, 4), tuple(xyz.shape)
    n, s = xyz.shape
    assert out_xyz.is_cuda and out_xyz.dtype == torch.float32 and out_xyz.is_contiguous() and out_xyz.numel() >= 3 * n
    assert out_index.is_cuda and out_index.dtype == torch.int32 and out_index.is_contiguous() and out_index.numel() >= n
    assert n_out.is_cuda and n_out.dtype == torch.int64 and n_out.numel() >= 1
    _check(lib().far_voxelize_static(_ptr(xyz), n, s, voxel, _ptr(out_xyz), _ptr(out_index), _ptr(n_out), _stream()),
           "far_voxelize_static")


def motion_fit(times, vel6, t_ref):
    """far_motion_fit (host-only FP64 helper, R15): returns (a, b) of xi(t) = a + b (t - t_ref)"""
    t = np.ascontiguousarray(times, dtype=np.float64)
    v = np.ascontiguousarray(vel6, dtype=np.float64).reshape(len(t), 6)
    m = Motion()
    _check(lib().far_motion_fit(C.c_void_p(t.ctypes.data), C.c_void_p(v.ctypes.data), len(t), float(t_ref), C.byref(m)),
           "far_motion_fit")
    return m.to_ab()


def undistort(xyz, time, dt_ref, a, b, out=None):
    """far_undistort (R16): device (n,3|4) points + device (n,) fp32 time offsets -> device (n,3)"""
    x, n, s = _points(xyz)
    t = time if isinstance(time, torch.Tensor) else torch.as_tensor(np.ascontiguousarray(time, dtype=np.float32))
    t = t.to(device="cuda", dtype=torch.float32).contiguous()
    assert t.shape == (n,)
    if out is None:
        out = torch.empty((n, 3), dtype=torch.float32, device="cuda")
    m = Motion.from_ab(a, b)
    _check(lib().far_undistort(_ptr(x), _ptr(t), n, s, float(dt_ref), C.byref(m), _ptr(out), _stream()), "far_undistort")
    return out


class Map:
    """A far_map_t handle.  All bulk arguments are CUDA tensors (NumPy arrays are uploaded for convenience)."""

    def __init__(self, voxel, cap, max_voxels, with_cov=False, k_cov=10, cov_eps=1e-3, max_load=0.5, max_batch=1 << 20,
                 renumber_every=0, min_spacing=0.0, _borrowed=None):
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2606_26010_b200 needs a CUDA device: there is no CPU fallback")
        self.voxel, self.cap, self.k_cov, self.with_cov = float(voxel), int(cap), int(k_cov), bool(with_cov)
        self._owned = _borrowed is None
        if _borrowed is None:
            cfg = MapConfig(voxel, cap, int(max_voxels), max_load, int(with_cov), k_cov, cov_eps, int(max_batch), int(renumber_every),
                            float(min_spacing))
            h = C.c_void_p()
            _check(lib().far_map_create(C.byref(h), C.byref(cfg)), "far_map_create")
            self._h = h
        else:
            self._h = _borrowed
        dev = torch.device("cuda", torch.cuda.current_device())
        self.device = dev
        self._insert_stats = torch.zeros(5, dtype=torch.int64, device=dev)
        self._prune_stats = torch.zeros(4, dtype=torch.int64, device=dev)
        self._map_stats = torch.zeros(len(MAP_STATS_FIELDS), dtype=torch.int64, device=dev)
        self.full_seen = False
        self._result = torch.zeros(GICP_RESULT_BYTES, dtype=torch.uint8, device=dev)

    def close(self):
        if getattr(self, "_h", None):
            if self._owned:
                lib().far_map_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- map maintenance ---------------------------------------------------------------------------
    def clear(self):
        _check(lib().far_map_clear(self._h, _stream()), "far_map_clear")

    def insert_enqueue(self, xyz, pose=None, compute_cov=False, d_pose=None):
        """far_map_insert / far_map_insert_dev without reading the statistics back (no host sync)."""
        x, n, s = _points(xyz)
        if d_pose is not None:
            rc = lib().far_map_insert_dev(self._h, _ptr(x), n, s, _ptr(d_pose), int(compute_cov), _ptr(self._insert_stats), _stream())
        else:
            pp = C.byref(Pose.from_rt(pose)) if pose is not None else None
            rc = lib().far_map_insert(self._h, _ptr(x), n, s, pp, int(compute_cov), _ptr(self._insert_stats), _stream())
        self.full_seen = _check(rc, "far_map_insert", full_ok=True)

    def insert(self, xyz, pose=None, compute_cov=False):
        self.insert_enqueue(xyz, pose, compute_cov)
        return dict(zip(INSERT_STATS_FIELDS, self._insert_stats.tolist()))

    def asmd_density(self, center, r_close, out=None):
        """far_asmd_density (R17): device double[2] = (n_close, number of close voxels)"""
        if out is None:
            out = torch.empty(2, dtype=torch.float64, device="cuda")
        c = (C.c_double * 3)(*[float(v) for v in center])
        _check(lib().far_asmd_density(self._h, c, float(r_close), _ptr(out), _stream()), "far_asmd_density")
        return out

    def insert_asmd_enqueue(self, xyz, d_n_close, d_max, pose=None, compute_cov=False, d_pose=None):
        """far_map_insert_asmd(_dev): per-voxel limit N_ASMD; d_n_close is a device double tensor"""
        x, n, s = _points(xyz)
        if not isinstance(d_n_close, torch.Tensor):
            d_n_close = torch.tensor([float(d_n_close)], dtype=torch.float64, device="cuda")
        if d_pose is not None:
            rc = lib().far_map_insert_asmd_dev(self._h, _ptr(x), n, s, _ptr(d_pose), _ptr(d_n_close), float(d_max),
                                               int(compute_cov), _ptr(self._insert_stats), _stream())
        else:
            pp = C.byref(Pose.from_rt(pose)) if pose is not None else None
            rc = lib().far_map_insert_asmd(self._h, _ptr(x), n, s, pp, _ptr(d_n_close), float(d_max), int(compute_cov),
                                           _ptr(self._insert_stats), _stream())
        self.full_seen = _check(rc, "far_map_insert_asmd", full_ok=True)
        self._keep = d_n_close

    def insert_asmd(self, xyz, n_close, d_max, pose=None, compute_cov=False):
        self.insert_asmd_enqueue(xyz, n_close, d_max, pose, compute_cov)
        return dict(zip(INSERT_STATS_FIELDS, self._insert_stats.tolist()))

    def prune_enqueue(self, center=None, radius=0.0, d_pose=None):
        if d_pose is not None:
            rc = lib().far_map_prune_dev(self._h, _ptr(d_pose), float(radius), _ptr(self._prune_stats), _stream())
        else:
            c = (C.c_double * 3)(*[float(v) for v in center])
            rc = lib().far_map_prune(self._h, c, float(radius), _ptr(self._prune_stats), _stream())
        _check(rc, "far_map_prune")

    def prune(self, center, radius):
        self.prune_enqueue(center, radius)
        return dict(zip(PRUNE_STATS_FIELDS, self._prune_stats.tolist()))

    def stats(self):
        _check(lib().far_map_stats(self._h, _ptr(self._map_stats), _stream()), "far_map_stats")
        return dict(zip(MAP_STATS_FIELDS, self._map_stats.tolist()))

    def size(self):
        s = self.stats()
        return s["n_voxels"], s["n_points"], s["next_id"]

    def snapshot(self):
        """far_map_snapshot_create: returns an opaque handle for restore()."""
        h = C.c_void_p()
        _check(lib().far_map_snapshot_create(self._h, C.byref(h), _stream()), "far_map_snapshot_create")
        return h

    def restore(self, snap):
        _check(lib().far_map_snapshot_restore(self._h, snap, _stream()), "far_map_snapshot_restore")

    @staticmethod
    def snapshot_destroy(snap):
        lib().far_map_snapshot_destroy(snap)

    def count27(self, q, with_voxels=False):
        """candidates in the 27 voxels around each query (and, optionally, how many of the 27 are occupied)"""
        x, n, s = _points(q)
        out = torch.empty(n, dtype=torch.int32, device=x.device)
        vox = torch.empty(n, dtype=torch.int32, device=x.device) if with_voxels else None
        _check(lib().far_map_count27(self._h, _ptr(x), n, s, _ptr(out), _ptr(vox), _stream()), "far_map_count27")
        return (out, vox) if with_voxels else out

    def rehash(self):
        _check(lib().far_map_rehash(self._h, _stream()), "far_map_rehash")

    def renumber(self):
        """far_map_renumber (R22): ids -= smallest live id; no host sync."""
        _check(lib().far_map_renumber(self._h, _stream()), "far_map_renumber")

    def status(self):
        """far_map_status: OK or ERR_FULL from the host-visible mirror of the device flag (never synchronises)."""
        return int(lib().far_map_status(self._h))

    def export(self, with_cov=False):
        """Live voxels sorted by key (the library's order is unspecified; sorting is presentation only)."""
        nv = self.stats()["n_voxels"]
        dev = self.device
        keys = torch.empty(max(nv, 1), dtype=torch.int64, device=dev)
        counts = torch.empty(max(nv, 1), dtype=torch.int32, device=dev)
        pts = torch.empty((max(nv, 1), self.cap, 4), dtype=torch.float32, device=dev)
        cov = torch.empty((max(nv, 1), self.cap, 6), dtype=torch.float32, device=dev) if with_cov else None
        cv = torch.empty((max(nv, 1), self.cap), dtype=torch.uint8, device=dev) if with_cov else None
        n_out = torch.zeros(1, dtype=torch.int64, device=dev)
        _check(lib().far_map_export(self._h, _ptr(keys), _ptr(counts), _ptr(pts), _ptr(cov), _ptr(cv), nv, _ptr(n_out),
                                    _stream()), "far_map_export")
        assert int(n_out.item()) == nv
        k = keys[:nv].cpu().numpy().view(np.uint64)
        order = np.argsort(k, kind="stable")
        p = pts[:nv].cpu().numpy()[order]
        out = dict(keys=k[order], counts=counts[:nv].cpu().numpy()[order], xyz=p[:, :, :3].copy(),
                   ids=p[:, :, 3].copy().view(np.uint32), cov=None, cov_valid=None)
        if with_cov:
            out["cov"] = cov[:nv].cpu().numpy()[order]
            out["cov_valid"] = cv[:nv].cpu().numpy()[order]
        return out

    # ---- queries -----------------------------------------------------------------------------------
    def nn(self, q, out_id=None, out_d2=None):
        """far_map_nn: (id int32-tensor holding uint32 bit patterns, d2 fp32) on the device."""
        x, n, s = _points(q)
        ids = out_id if out_id is not None else torch.empty(n, dtype=torch.int32, device=x.device)
        d2 = out_d2 if out_d2 is not None else torch.empty(n, dtype=torch.float32, device=x.device)
        _check(lib().far_map_nn(self._h, _ptr(x), n, s, _ptr(ids), _ptr(d2), _stream()), "far_map_nn")
        return ids, d2

    def knn_cov(self, q, out_cov=None, out_valid=None, d_m=None):
        x, n, s = _points(q)
        cov = out_cov if out_cov is not None else torch.empty((n, 6), dtype=torch.float32, device=x.device)
        valid = out_valid if out_valid is not None else torch.empty(n, dtype=torch.uint8, device=x.device)
        if d_m is not None:
            rc = lib().far_map_knn_cov_dev(self._h, _ptr(x), _ptr(d_m), n, s, _ptr(cov), _ptr(valid), _stream())
        else:
            rc = lib().far_map_knn_cov(self._h, _ptr(x), n, s, _ptr(cov), _ptr(valid), _stream())
        _check(rc, "far_map_knn_cov")
        return cov, valid

    # ---- GICP --------------------------------------------------------------------------------------
    def _scan_args(self, scan, cov6, valid):
        x, n, s = _points(scan)
        if cov6 is not None and not isinstance(cov6, torch.Tensor):
            cov6 = torch.as_tensor(np.ascontiguousarray(cov6, dtype=np.float32)).to(x.device)
        if valid is not None and not isinstance(valid, torch.Tensor):
            valid = torch.as_tensor(np.ascontiguousarray(valid, dtype=np.uint8)).to(x.device)
        return x, n, s, cov6, valid

    def gicp_linearize(self, scan, cov6, valid, pose, sigma, opts=None):
        x, n, s, c, v = self._scan_args(scan, cov6, valid)
        po = Pose.from_rt(pose)
        _check(lib().far_gicp_linearize(self._h, _ptr(x), _ptr(c), _ptr(v), n, s, C.byref(po), float(sigma),
                                        C.byref(opts) if opts is not None else None, _ptr(self._result), _stream()),
               "far_gicp_linearize")
        return result_to_dict(_struct_from_tensor(self._result, GicpResult))

    def gicp_register_enqueue(self, scan, cov6, valid, init_pose, sigma, max_iters=30, opts=None, d_n=None, d_init_pose=None,
                              d_result=None):
        """far_gicp_register(_dev): enqueue only; the result struct stays on the device (self._result or d_result)."""
        x, n, s, c, v = self._scan_args(scan, cov6, valid)
        res = d_result if d_result is not None else self._result
        o = C.byref(opts) if opts is not None else None
        if d_n is not None:
            rc = lib().far_gicp_register_dev(self._h, _ptr(x), _ptr(c), _ptr(v), _ptr(d_n), n, s, _ptr(d_init_pose), float(sigma),
                                             int(max_iters), o, _ptr(res), _stream())
        else:
            po = Pose.from_rt(init_pose)
            rc = lib().far_gicp_register(self._h, _ptr(x), _ptr(c), _ptr(v), n, s, C.byref(po), float(sigma), int(max_iters),
                                         o, _ptr(res), _stream())
        _check(rc, "far_gicp_register")
        return res

    def gicp_register(self, scan, cov6, valid, init_pose, sigma, max_iters=30, opts=None):
        res = self.gicp_register_enqueue(scan, cov6, valid, init_pose, sigma, max_iters, opts)
        return result_to_dict(_struct_from_tensor(res, GicpResult))


class Frontend:
    """far_frontend_*: one frame through the whole hot path as a single stream-ordered chain."""

    def __init__(self, voxel, cap, max_voxels, max_scan_points, ds_voxel=0.0, prune_radius=0.0, max_iters=30,
                 update_map=True, opts=None, k_cov=10, cov_eps=1e-3, max_load=0.5, asmd=False, asmd_r_close=10.0,
                 asmd_d_max=100.0, use_graph=True, min_spacing=0.0):
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2606_26010_b200 needs a CUDA device: there is no CPU fallback")
        o = opts if opts is not None else default_options()
        cfg = FrontendConfig(MapConfig(voxel, cap, int(max_voxels), max_load, 1, k_cov, cov_eps, 0, 0, float(min_spacing)), ds_voxel,
                             int(max_scan_points), float(prune_radius), int(max_iters), int(update_map), o,
                             int(asmd), float(asmd_r_close), float(asmd_d_max), int(use_graph))
        h = C.c_void_p()
        _check(lib().far_frontend_create(C.byref(h), C.byref(cfg)), "far_frontend_create")
        self._h = h
        self.map = Map(voxel, cap, max_voxels, with_cov=True, k_cov=k_cov, _borrowed=C.c_void_p(lib().far_frontend_map(h)))
        self.max_scan_points = int(max_scan_points)
        self.h_result = GicpResult()
        self.full_seen = False

    def close(self):
        if getattr(self, "_h", None):
            self.map.close()
            lib().far_frontend_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def process_enqueue(self, d_scan, init_pose, sigma, d_result=None):
        """Device scan in, result struct stays on the device; no host synchronisation."""
        x, n, s = _points(d_scan)
        po = Pose.from_rt(init_pose) if not isinstance(init_pose, Pose) else init_pose
        self.full_seen = _check(lib().far_frontend_process(self._h, _ptr(x), n, s, C.byref(po), float(sigma), _ptr(d_result),
                                                           _stream()), "far_frontend_process", full_ok=True)

    def process_sweep_enqueue(self, d_scan, d_time, dt_ref, a, b, init_pose, sigma, d_result=None):
        """Raw sweep + per-point time offsets in: far_undistort, then the chain of process_enqueue."""
        x, n, s = _points(d_scan)
        assert d_time.dtype == torch.float32 and d_time.shape == (n,) and d_time.is_cuda
        po = Pose.from_rt(init_pose) if not isinstance(init_pose, Pose) else init_pose
        m = Motion.from_ab(a, b)
        self.full_seen = _check(lib().far_frontend_process_sweep(self._h, _ptr(x), _ptr(d_time), n, s, float(dt_ref), C.byref(m),
                                                                 C.byref(po), float(sigma), _ptr(d_result), _stream()),
                                "far_frontend_process_sweep", full_ok=True)

    def process_host(self, h_scan, init_pose, sigma):
        """HOST scan (a pinned torch CPU tensor or a NumPy array) in, result dict out; uploads, runs, downloads, syncs."""
        if isinstance(h_scan, torch.Tensor):
            assert h_scan.device.type == "cpu" and h_scan.dtype == torch.float32 and h_scan.is_contiguous()
            ptr, n, s = C.c_void_p(h_scan.data_ptr()), h_scan.shape[0], h_scan.shape[1]
        else:
            h_scan = np.ascontiguousarray(h_scan, dtype=np.float32)
            ptr, n, s = C.c_void_p(h_scan.ctypes.data), h_scan.shape[0], h_scan.shape[1]
        po = Pose.from_rt(init_pose) if not isinstance(init_pose, Pose) else init_pose
        self.full_seen = _check(lib().far_frontend_process_host(self._h, ptr, n, s, C.byref(po), float(sigma),
                                                                C.byref(self.h_result), _stream()),
                                "far_frontend_process_host", full_ok=True)
        return result_to_dict(self.h_result)

    def graph_state(self):
        """far_frontend_graph_state: 1 replaying the captured frame graph, 0 not captured yet, -1 capture refused"""
        return int(lib().far_frontend_graph_state(self._h))

    def insert_stats(self):
        """far_frontend_insert_stats: statistics of the last frame's map update (synchronising read of the device struct)."""
        buf = (C.c_int64 * 5)()
        _check(lib().far_frontend_insert_stats(self._h, buf, _stream()), "far_frontend_insert_stats")
        return dict(zip(INSERT_STATS_FIELDS, list(buf)))


def _dp(a):
    return C.c_void_p(a.ctypes.data) if a is not None else None


def lidar_velocity(T_t, T_prev, dt):
    """far_lidar_velocity (Eq. 7)"""
    v = np.zeros(3)
    _check(lib().far_lidar_velocity(C.byref(Pose.from_rt(T_t)), C.byref(Pose.from_rt(T_prev)), float(dt), _dp(v)), "far_lidar_velocity")
    return v


def ekf_model(x, u, dt):
    """far_ekf_model: Eq. 9 step and its analytic Jacobian"""
    x = np.ascontiguousarray(x, dtype=np.float64); u = np.ascontiguousarray(u, dtype=np.float64)
    xn, F = np.zeros(9), np.zeros((9, 9))
    _check(lib().far_ekf_model(_dp(x), _dp(u), float(dt), _dp(xn), _dp(F)), "far_ekf_model")
    return xn, F


class Ekf:
    """far_ekf_*: host-only FP64 Sensor Fusion backend (Eq. 8-11; R18-R20)"""

    def __init__(self, x0, P0_diag, Q_diag, dt=0.01, n_up=1, accel_bias=None, gyro_bias=None):
        a = [np.ascontiguousarray(v, dtype=np.float64) for v in (x0, P0_diag, Q_diag)]
        ab = np.ascontiguousarray(accel_bias, dtype=np.float64) if accel_bias is not None else None
        wb = np.ascontiguousarray(gyro_bias, dtype=np.float64) if gyro_bias is not None else None
        self._h = lib().far_ekf_create(_dp(a[0]), _dp(a[1]), _dp(a[2]), float(dt), int(n_up), _dp(ab), _dp(wb))
        if not self._h:
            raise ValueError("bad EKF configuration")
        self.dt = float(dt)

    def __del__(self):
        if getattr(self, "_h", None) and lib is not None and _lib is not None:     # not during interpreter teardown
            _lib.far_ekf_destroy(self._h)
            self._h = None

    def predict(self, accel_m, gyro_m):
        a = np.ascontiguousarray(accel_m, dtype=np.float64); w = np.ascontiguousarray(gyro_m, dtype=np.float64)
        return int(lib().far_ekf_predict(self._h, _dp(a), _dp(w)))

    def push_lidar(self, T_L, v_L, R_diag, cycle_s, theta_ref=None):
        v = np.ascontiguousarray(v_L, dtype=np.float64); r = np.ascontiguousarray(R_diag, dtype=np.float64)
        tr = np.ascontiguousarray(theta_ref, dtype=np.float64) if theta_ref is not None else None
        assert len(r) == (11 if tr is not None else 9)
        _check(lib().far_ekf_push_lidar(self._h, C.byref(Pose.from_rt(T_L)), _dp(v), _dp(tr), _dp(r), int(cycle_s)), "far_ekf_push_lidar")

    def state(self):
        x, P, k = np.zeros(9), np.zeros((9, 9)), C.c_int64(0)
        _check(lib().far_ekf_state(self._h, _dp(x), _dp(P), C.byref(k)), "far_ekf_state")
        return x, P, k.value

    def pose(self):
        p = Pose()
        _check(lib().far_ekf_pose(self._h, C.byref(p)), "far_ekf_pose")
        return p.to_rt()

    def velocity_history(self, m):
        t, v = np.zeros(m), np.zeros((m, 6))
        n = lib().far_ekf_velocity_history(self._h, int(m), _dp(t), _dp(v))
        return t[:n], v[:n]


class AdaptiveThreshold:
    """far_threshold_*: host-side sigma of the adaptive correspondence threshold."""

    def __init__(self, sigma0=2.0, min_motion=0.1, max_range=100.0):
        self._h = C.c_void_p(lib().far_threshold_create(sigma0, min_motion, max_range))

    def __del__(self):
        if getattr(self, "_h", None) and lib is not None and _lib is not None:     # not during interpreter teardown
            _lib.far_threshold_destroy(self._h)
            self._h = None

    def update(self, predicted, registered):
        a, b = Pose.from_rt(predicted), Pose.from_rt(registered)
        lib().far_threshold_update(self._h, C.byref(a), C.byref(b))

    def sigma(self):
        return lib().far_threshold_sigma(self._h)
