"""ORACLE (test infrastructure, not the product): ctypes binding of oracle/libfaro.so.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It never imports paper_2606_26010_b200 and shares no code with it.
All arrays are NumPy host arrays.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

_HERE = os.path.dirname(os.path.abspath(__file__))
NO_ID = 0xFFFFFFFF
KERNEL_CAUCHY, KERNEL_GEMAN_MCCLURE, KERNEL_NONE = 0, 1, 2
OK, ERR_ARG, ERR_RANGE, ERR_DEGENERATE = 0, 1, 4, 5


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


class InsertStats(C.Structure):
    _fields_ = [(n, C.c_int64) for n in ("n_offered", "n_accepted", "n_new_voxels", "n_dropped_full", "n_invalid")]


class PruneStats(C.Structure):
    _fields_ = [(n, C.c_int64) for n in ("n_voxels_removed", "n_points_removed", "n_voxels_left", "n_points_left")]


class Motion(C.Structure):
    """xi(t) = a + b (t - t_ref): body twist, linear velocity first (R15)"""
    _fields_ = [("a", C.c_double * 6), ("b", C.c_double * 6)]

    @staticmethod
    def from_ab(a, b):
        m = Motion()
        m.a[:] = np.asarray(a, dtype=np.float64).reshape(6).tolist()
        m.b[:] = np.asarray(b, dtype=np.float64).reshape(6).tolist()
        return m

    def to_ab(self):
        return np.array(self.a[:]), np.array(self.b[:])


class GicpOptions(C.Structure):
    _fields_ = [("kernel", C.c_int32), ("conv_eps", C.c_double), ("tau_mult", C.c_double), ("kappa_div", C.c_double)]


class GicpResult(C.Structure):
    _fields_ = [("pose", Pose), ("H", C.c_double * 36), ("b", C.c_double * 6), ("chi2", C.c_double),
                ("n_inliers", C.c_int32), ("iters", C.c_int32), ("converged", C.c_int32), ("status", C.c_int32)]

    def as_dict(self):
        R, t = self.pose.to_rt()
        return dict(R=R, t=t, H=np.array(self.H[:]).reshape(6, 6), b=np.array(self.b[:]), chi2=self.chi2,
                    n_inliers=self.n_inliers, iters=self.iters, converged=self.converged, status=self.status)


_lib = None


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        vp, i64, i32, f32, f64 = C.c_void_p, C.c_int64, C.c_int32, C.c_float, C.c_double
        L.faro_map_create.restype = vp
        L.faro_map_create.argtypes = [f32, i32, i32, f64]
        L.faro_map_destroy.argtypes = [vp]
        L.faro_map_destroy.restype = None
        L.faro_map_clone.restype = vp
        L.faro_map_clone.argtypes = [vp]
        L.faro_pack_key.restype = C.c_uint64
        L.faro_pack_key.argtypes = [i32, i32, i32]
        L.faro_unpack_key.restype = None
        L.faro_unpack_key.argtypes = [C.c_uint64, vp]
        L.faro_keys.argtypes = [vp, i64, C.c_int, f32, vp, vp]
        L.faro_voxelize.argtypes = [vp, i64, C.c_int, f32, vp, vp, vp]
        L.faro_map_insert.argtypes = [vp, vp, i64, C.c_int, vp, C.c_int, vp]
        L.faro_map_prune.argtypes = [vp, vp, f64, vp]
        L.faro_map_size.argtypes = [vp, vp, vp, vp]
        L.faro_map_renumber.argtypes = [vp, vp]
        L.faro_map_set_min_spacing.argtypes = [vp, f64]
        L.faro_map_set_min_spacing.restype = None
        L.faro_map_export.argtypes = [vp, vp, vp, vp, vp, vp]
        L.faro_map_nn.argtypes = [vp, vp, i64, C.c_int, vp, vp, C.c_int]
        L.faro_map_nn_brute.argtypes = [vp, vp, i64, C.c_int, vp, vp]
        L.faro_map_knn.argtypes = [vp, vp, i64, C.c_int, i32, vp, vp]
        L.faro_map_knn_cov.argtypes = [vp, vp, i64, C.c_int, vp, vp, C.c_int]
        L.faro_cov_from_points.argtypes = [vp, i32, C.c_int, f64, vp]
        L.faro_gicp_linearize.argtypes = [vp, vp, vp, vp, i64, C.c_int, vp, f64, vp, vp, C.c_int]
        L.faro_gicp_register.argtypes = [vp, vp, vp, vp, i64, C.c_int, vp, f64, C.c_int, vp, vp, C.c_int]
        L.faro_gicp_correspondences.argtypes = [vp, vp, vp, vp, i64, C.c_int, vp, f64, vp, vp, vp, vp, vp, vp, vp]
        L.faro_gicp_default_options.argtypes = [vp]
        L.faro_gicp_default_options.restype = None
        L.faro_se3_exp.argtypes = [vp, vp]
        L.faro_se3_exp.restype = None
        L.faro_robust_weight.argtypes = [C.c_int, f64, f64]
        L.faro_robust_weight.restype = f64
        L.faro_threshold_create.restype = vp
        L.faro_threshold_create.argtypes = [f64, f64, f64]
        L.faro_threshold_destroy.argtypes = [vp]
        L.faro_threshold_destroy.restype = None
        L.faro_threshold_update.argtypes = [vp, vp, vp]
        L.faro_threshold_update.restype = None
        L.faro_threshold_sigma.argtypes = [vp]
        L.faro_threshold_sigma.restype = f64
        L.faro_motion_fit.argtypes = [vp, vp, i32, f64, vp]
        L.faro_undistort.argtypes = [vp, vp, i64, C.c_int, f64, vp, vp]
        L.faro_asmd_density.argtypes = [vp, vp, f64, vp, vp]
        L.faro_asmd_cap.argtypes = [vp, f32, vp, f64, f64, i32, i32]
        L.faro_asmd_cap.restype = i32
        L.faro_map_insert_asmd.argtypes = [vp, vp, i64, C.c_int, vp, f64, f64, C.c_int, vp]
        _lib = L
    return _lib


def _pts(a):
    a = np.ascontiguousarray(a, dtype=np.float32)
    assert a.ndim == 2 and a.shape[1] in (3, 4), a.shape
    return a, a.shape[0], a.shape[1]


def _p(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


def _check(rc):
    if rc != 0:
        raise RuntimeError(f"oracle call failed with status {rc}")


def default_options(kernel=KERNEL_CAUCHY, conv_eps=5e-3, tau_mult=3.0, kappa_div=3.0):
    return GicpOptions(kernel, conv_eps, tau_mult, kappa_div)


def pack_key(kx, ky, kz):
    return int(lib().faro_pack_key(int(kx), int(ky), int(kz)))


def unpack_key(key):
    k = np.zeros(3, dtype=np.int32)
    lib().faro_unpack_key(C.c_uint64(int(key)), _p(k))
    return k


def keys(xyz, voxel):
    a, n, s = _pts(xyz)
    k = np.empty(n, dtype=np.uint64)
    v = np.empty(n, dtype=np.uint8)
    _check(lib().faro_keys(_p(a), n, s, voxel, _p(k), _p(v)))
    return k, v.astype(bool)


def voxelize(xyz, voxel):
    a, n, s = _pts(xyz)
    out = np.empty((n, 3), dtype=np.float32)
    idx = np.empty(n, dtype=np.int32)
    m = C.c_int64(0)
    _check(lib().faro_voxelize(_p(a), n, s, voxel, _p(out), _p(idx), C.byref(m)))
    return out[:m.value].copy(), idx[:m.value].copy()


def se3_exp(delta):
    d = np.ascontiguousarray(delta, dtype=np.float64)
    p = Pose()
    lib().faro_se3_exp(_p(d), C.byref(p))
    return p.to_rt()


def robust_weight(kernel, e2, kappa):
    return lib().faro_robust_weight(kernel, e2, kappa)


def cov_from_points(pts, eps=1e-3):
    a, n, s = _pts(pts)
    out = np.empty(6, dtype=np.float64)
    _check(lib().faro_cov_from_points(_p(a), n, s, eps, _p(out)))
    return out


def motion_fit(times, vel6, t_ref):
    """R15: least-squares line per twist component over the velocity history; returns (a, b)"""
    t = np.ascontiguousarray(times, dtype=np.float64)
    v = np.ascontiguousarray(vel6, dtype=np.float64).reshape(len(t), 6)
    m = Motion()
    _check(lib().faro_motion_fit(_p(t), _p(v), len(t), float(t_ref), C.byref(m)))
    return m.to_ab()


def undistort(xyz, time, dt_ref, a, b):
    """R16: every point projected to the frame reference timestamp"""
    p, n, s = _pts(xyz)
    t = np.ascontiguousarray(time, dtype=np.float32)
    assert t.shape == (n,)
    out = np.empty((n, 3), dtype=np.float32)
    m = Motion.from_ab(a, b)
    _check(lib().faro_undistort(_p(p), _p(t), n, s, float(dt_ref), C.byref(m), _p(out)))
    return out


def asmd_cap(k3, voxel, center, n_close, d_max, k_min, cap):
    k = np.ascontiguousarray(k3, dtype=np.int32)
    c = np.ascontiguousarray(center, dtype=np.float64)
    return int(lib().faro_asmd_cap(_p(k), voxel, _p(c), float(n_close), float(d_max), int(k_min), int(cap)))


class Map:
    def __init__(self, voxel, cap, k_cov=10, cov_eps=1e-3, min_spacing=0.0):
        self.voxel, self.cap, self.k_cov = float(voxel), int(cap), int(k_cov)
        self._h = lib().faro_map_create(voxel, cap, k_cov, cov_eps)
        if not self._h:
            raise ValueError("bad map config")
        if min_spacing > 0.0:
            lib().faro_map_set_min_spacing(self._h, float(min_spacing))

    def __del__(self):
        if getattr(self, "_h", None):
            lib().faro_map_destroy(self._h)
            self._h = None

    def clone(self):
        """faro_map_clone: an independent deep copy (contents, covariances, id counter, configuration)."""
        c = Map.__new__(Map)
        c.voxel, c.cap, c.k_cov = self.voxel, self.cap, self.k_cov
        c._h = lib().faro_map_clone(self._h)
        if not c._h:
            raise MemoryError("faro_map_clone")
        return c

    def insert(self, xyz, pose=None, compute_cov=False):
        a, n, s = _pts(xyz)
        st = InsertStats()
        pp = C.byref(Pose.from_rt(pose)) if pose is not None else None
        _check(lib().faro_map_insert(self._h, _p(a), n, s, pp, int(compute_cov), C.byref(st)))
        return {f: getattr(st, f) for f, _ in st._fields_}

    def insert_asmd(self, xyz, n_close, d_max, pose=None, compute_cov=False):
        """PAPER.md:109 / R17: per-voxel limit N_ASMD instead of the fixed cap"""
        a, n, s = _pts(xyz)
        st = InsertStats()
        pp = C.byref(Pose.from_rt(pose)) if pose is not None else None
        _check(lib().faro_map_insert_asmd(self._h, _p(a), n, s, pp, float(n_close), float(d_max), int(compute_cov),
                                          C.byref(st)))
        return {f: getattr(st, f) for f, _ in st._fields_}

    def asmd_density(self, center, r_close):
        """mean stored points per voxel within r_close of center, and the number of such voxels"""
        c = np.ascontiguousarray(center, dtype=np.float64)
        out, nv = C.c_double(0.0), C.c_int64(0)
        _check(lib().faro_asmd_density(self._h, _p(c), float(r_close), C.byref(out), C.byref(nv)))
        return out.value, nv.value

    def prune(self, center, radius):
        c = np.ascontiguousarray(center, dtype=np.float64)
        st = PruneStats()
        _check(lib().faro_map_prune(self._h, _p(c), float(radius), C.byref(st)))
        return {f: getattr(st, f) for f, _ in st._fields_}

    def size(self):
        nv, npnt, nid = C.c_int64(), C.c_int64(), C.c_uint64()
        _check(lib().faro_map_size(self._h, C.byref(nv), C.byref(npnt), C.byref(nid)))
        return nv.value, npnt.value, nid.value

    def renumber(self):
        """R22: ids -= smallest stored id; returns what was subtracted"""
        sub = C.c_uint64()
        _check(lib().faro_map_renumber(self._h, C.byref(sub)))
        return sub.value

    def export(self, with_cov=False):
        nv = self.size()[0]
        keys_ = np.empty(nv, dtype=np.uint64)
        counts = np.empty(nv, dtype=np.int32)
        pts = np.empty((nv, self.cap, 4), dtype=np.float32)
        cov = np.empty((nv, self.cap, 6), dtype=np.float32) if with_cov else None
        cv = np.empty((nv, self.cap), dtype=np.uint8) if with_cov else None
        _check(lib().faro_map_export(self._h, _p(keys_), _p(counts), _p(pts), _p(cov), _p(cv)))
        ids = pts[:, :, 3].copy().view(np.uint32)
        return dict(keys=keys_, counts=counts, xyz=pts[:, :, :3].copy(), ids=ids, cov=cov, cov_valid=cv)

    def nn(self, q, nthreads=1):
        a, n, s = _pts(q)
        ids = np.empty(n, dtype=np.uint32)
        d2 = np.empty(n, dtype=np.float32)
        _check(lib().faro_map_nn(self._h, _p(a), n, s, _p(ids), _p(d2), nthreads))
        return ids, d2

    def nn_brute(self, q):
        a, n, s = _pts(q)
        ids = np.empty(n, dtype=np.uint32)
        d2 = np.empty(n, dtype=np.float32)
        _check(lib().faro_map_nn_brute(self._h, _p(a), n, s, _p(ids), _p(d2)))
        return ids, d2

    def knn(self, q, k):
        a, n, s = _pts(q)
        ids = np.empty((n, k), dtype=np.uint32)
        d2 = np.empty((n, k), dtype=np.float64)
        _check(lib().faro_map_knn(self._h, _p(a), n, s, k, _p(ids), _p(d2)))
        return ids, d2

    def knn_cov(self, q, nthreads=1):
        a, n, s = _pts(q)
        cov = np.empty((n, 6), dtype=np.float32)
        valid = np.empty(n, dtype=np.uint8)
        _check(lib().faro_map_knn_cov(self._h, _p(a), n, s, _p(cov), _p(valid), nthreads))
        return cov, valid

    def _scan_args(self, scan, cov6, valid):
        a, n, s = _pts(scan)
        c = np.ascontiguousarray(cov6, dtype=np.float32) if cov6 is not None else None
        v = np.ascontiguousarray(valid, dtype=np.uint8) if valid is not None else None
        return a, n, s, c, v

    def gicp_linearize(self, scan, cov6, valid, pose, sigma, opts=None, nthreads=1):
        a, n, s, c, v = self._scan_args(scan, cov6, valid)
        res = GicpResult()
        po = Pose.from_rt(pose)
        _check(lib().faro_gicp_linearize(self._h, _p(a), _p(c), _p(v), n, s, C.byref(po), float(sigma),
                                         C.byref(opts) if opts is not None else None, C.byref(res), nthreads))
        return res.as_dict()

    def gicp_register(self, scan, cov6, valid, init_pose, sigma, max_iters=30, opts=None, nthreads=1):
        a, n, s, c, v = self._scan_args(scan, cov6, valid)
        res = GicpResult()
        po = Pose.from_rt(init_pose)
        _check(lib().faro_gicp_register(self._h, _p(a), _p(c), _p(v), n, s, C.byref(po), float(sigma), int(max_iters),
                                        C.byref(opts) if opts is not None else None, C.byref(res), nthreads))
        return res.as_dict()

    def gicp_correspondences(self, scan, cov6, valid, pose, sigma, opts=None):
        a, n, s, c, v = self._scan_args(scan, cov6, valid)
        used = np.empty(n, dtype=np.uint8)
        p3 = np.empty((n, 3)); r3 = np.empty((n, 3)); M9 = np.empty((n, 3, 3)); w = np.empty(n)
        ids = np.empty(n, dtype=np.uint32)
        po = Pose.from_rt(pose)
        _check(lib().faro_gicp_correspondences(self._h, _p(a), _p(c), _p(v), n, s, C.byref(po), float(sigma),
                                               C.byref(opts) if opts is not None else None,
                                               _p(used), _p(p3), _p(r3), _p(M9), _p(w), _p(ids)))
        return dict(used=used.astype(bool), p=p3, r=r3, M=M9, w=w, id=ids)


class AdaptiveThreshold:
    def __init__(self, sigma0=2.0, min_motion=0.1, max_range=100.0):
        self._h = lib().faro_threshold_create(sigma0, min_motion, max_range)

    def __del__(self):
        if getattr(self, "_h", None):
            lib().faro_threshold_destroy(self._h)
            self._h = None

    def update(self, predicted, registered):
        a, b = Pose.from_rt(predicted), Pose.from_rt(registered)
        lib().faro_threshold_update(self._h, C.byref(a), C.byref(b))

    def sigma(self):
        return lib().faro_threshold_sigma(self._h)
