"""Seeded synthetic LiDAR-shaped inputs (NumPy only, fp32 outputs).

Nothing in this file belongs to the method under test: it makes points, poses
and scans.  Ray casting is analytic (planes, axis-aligned boxes via slabs,
vertical cylinders) -- compute only, no renderer.

Shapes follow the paper's workloads (HDL-64/OS1-64 style
64 x 2048 spinning scans of <100k returns; three long-range forward LiDARs of
~200k points per concatenated scan at up to 250 km/h) and BASELINE.json
configs C1..C5; the concrete recipes are those of SURVEY.md section 8(d).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

F32 = np.float32


# --------------------------------------------------------------------------
# poses: (R, t) with R 3x3 float64 row-major, t float64[3]; map_from_sensor
# --------------------------------------------------------------------------
def pose_identity():
    return np.eye(3), np.zeros(3)


def _rot_axis_angle(axis, angle):
    axis = np.asarray(axis, dtype=np.float64)
    axis = axis / np.linalg.norm(axis)
    K = np.array([[0, -axis[2], axis[1]], [axis[2], 0, -axis[0]], [-axis[1], axis[0], 0]])
    return np.eye(3) + math.sin(angle) * K + (1.0 - math.cos(angle)) * (K @ K)


def pose_from_rpy_t(roll, pitch, yaw, t):
    """ZYX Euler angles (radians) and translation."""
    Rz = _rot_axis_angle([0, 0, 1], yaw)
    Ry = _rot_axis_angle([0, 1, 0], pitch)
    Rx = _rot_axis_angle([1, 0, 0], roll)
    return Rz @ Ry @ Rx, np.asarray(t, dtype=np.float64).copy()


def pose_inverse(T):
    R, t = T
    return R.T.copy(), -(R.T @ t)


def pose_compose(A, B):
    """A * B (apply B first)."""
    return A[0] @ B[0], A[0] @ B[1] + A[1]


def pose_apply(T, pts):
    """Apply pose to an (N,3) array in float64 and return float32."""
    R, t = T
    return (np.asarray(pts, dtype=np.float64) @ R.T + t).astype(F32)


def perturb_pose(T, dtrans, drot_deg, rng):
    """Left-multiply T by a random rigid motion of given magnitude."""
    d = rng.normal(size=3)
    d = d / np.linalg.norm(d) * dtrans
    ax = rng.normal(size=3)
    Rp = _rot_axis_angle(ax, math.radians(drot_deg))
    # rotate about the sensor position so that the translation error is dtrans
    R, t = T
    return Rp @ R, t + d


# --------------------------------------------------------------------------
# C1: tiny three-plane scene
# --------------------------------------------------------------------------
def _c1_planes(n, rng):
    """Point i lies on plane (i mod 3): ground z=0, wall x=5, wall y=5."""
    u = rng.uniform(-5.0, 5.0, size=n)
    w = rng.uniform(-5.0, 5.0, size=n)
    h = rng.uniform(0.0, 3.0, size=n)
    which = np.arange(n) % 3
    pts = np.empty((n, 3), dtype=np.float64)
    g = which == 0
    pts[g] = np.stack([u[g], w[g], np.zeros(g.sum())], axis=1)
    a = which == 1
    pts[a] = np.stack([np.full(a.sum(), 5.0), u[a], h[a]], axis=1)
    b = which == 2
    pts[b] = np.stack([u[b], np.full(b.sum(), 5.0), h[b]], axis=1)
    return pts


def c1_tiny(seed=0, n_map=4096, n_scan=1024, noise=0.01, noise_free=False):
    """BASELINE.json configs[0].

    Returns dict(map_points f32[n_map,3], scan f32[n_scan,3] in the sensor frame,
    T_gt (map_from_sensor ground truth), T_init (identity), voxel, cap, sigma).
    Ground truth offset: yaw 2 deg, t = (0.2, -0.2, 0.1), |t| = 0.3 m.
    """
    rng = np.random.default_rng(seed)
    map_pts = _c1_planes(n_map, rng).astype(F32)
    T_gt = pose_from_rpy_t(0.0, 0.0, math.radians(2.0), [0.2, -0.2, 0.1])
    if noise_free:
        sel = rng.permutation(n_map)[:n_scan]
        world = map_pts[sel].astype(np.float64)
    else:
        world = _c1_planes(n_scan, rng) + rng.normal(0.0, noise, size=(n_scan, 3))
    scan = pose_apply(pose_inverse(T_gt), world)
    return dict(map_points=map_pts, scan=scan, T_gt=T_gt, T_init=pose_identity(),
                voxel=0.5, cap=20, sigma=2.0, max_iters=30)


# --------------------------------------------------------------------------
# Urban scene: ground plane, axis-aligned boxes, vertical cylinder poles
# --------------------------------------------------------------------------
@dataclass
class UrbanScene:
    seed: int = 1
    extent: float = 400.0      # square side [m], centred on the origin
    n_boxes: int = 300
    n_poles: int = 200
    street_half_width: float = 10.0
    pole_radius: float = 0.15
    pole_height: float = 8.0
    boxes: np.ndarray = field(init=False)   # (B,5): cx, cy, sx, sy, h
    poles: np.ndarray = field(init=False)   # (P,2): cx, cy

    def __post_init__(self):
        rng = np.random.default_rng(self.seed)
        half = self.extent / 2.0
        boxes = []
        while len(boxes) < self.n_boxes:
            m = 4 * self.n_boxes
            c = rng.uniform(-half, half, size=(m, 2))
            s = rng.uniform(5.0, 30.0, size=(m, 2))
            h = rng.uniform(5.0, 30.0, size=m)
            ok = np.abs(c[:, 1]) - s[:, 1] / 2.0 > self.street_half_width
            for i in np.nonzero(ok)[0]:
                boxes.append((c[i, 0], c[i, 1], s[i, 0], s[i, 1], h[i]))
                if len(boxes) == self.n_boxes:
                    break
        self.boxes = np.array(boxes, dtype=np.float64)
        px = rng.uniform(-half, half, size=self.n_poles)
        side = rng.choice([-1.0, 1.0], size=self.n_poles)
        py = side * rng.uniform(self.street_half_width - 3.0, self.street_half_width - 0.5,
                                size=self.n_poles)
        self.poles = np.stack([px, py], axis=1)

    # ---- ray casting ----------------------------------------------------
    def raycast(self, origin, dirs, chunk=4096, max_range=None):
        """Smallest positive hit distance along unit `dirs` from `origin`; inf if none.

        `max_range` only culls objects that cannot be hit within that range."""
        origin = np.asarray(origin, dtype=np.float64)
        dirs = np.asarray(dirs, dtype=np.float64)
        out = np.full(dirs.shape[0], np.inf)
        boxes, poles = self.boxes, self.poles
        if max_range is not None:
            bd = np.hypot(boxes[:, 0] - origin[0], boxes[:, 1] - origin[1]) - 0.5 * np.hypot(boxes[:, 2], boxes[:, 3])
            boxes = boxes[bd <= max_range + 1.0]
            pd = np.hypot(poles[:, 0] - origin[0], poles[:, 1] - origin[1])
            poles = poles[pd <= max_range + 1.0]
        lo = np.stack([boxes[:, 0] - boxes[:, 2] / 2, boxes[:, 1] - boxes[:, 3] / 2,
                       np.zeros(len(boxes))], axis=1)
        hi = np.stack([boxes[:, 0] + boxes[:, 2] / 2, boxes[:, 1] + boxes[:, 3] / 2,
                       boxes[:, 4]], axis=1)
        for s in range(0, dirs.shape[0], chunk):
            d = dirs[s:s + chunk]
            t = np.full(d.shape[0], np.inf)
            # ground z = 0
            with np.errstate(divide="ignore", invalid="ignore"):
                tg = -origin[2] / d[:, 2]
            tg[~(tg > 1e-6)] = np.inf
            t = np.minimum(t, tg)
            # boxes (slab method)
            with np.errstate(divide="ignore", invalid="ignore"):
                inv = 1.0 / d                                    # (n,3)
                t0 = (lo[None, :, :] - origin[None, None, :]) * inv[:, None, :]
                t1 = (hi[None, :, :] - origin[None, None, :]) * inv[:, None, :]
            tn = np.nanmax(np.minimum(t0, t1), axis=2)
            tf = np.nanmin(np.maximum(t0, t1), axis=2)
            hit = (tn <= tf) & (tf > 1e-6)
            tb = np.where(hit, np.where(tn > 1e-6, tn, tf), np.inf)
            t = np.minimum(t, tb.min(axis=1))
            # poles: vertical cylinders, side surface only
            ox = origin[0] - poles[:, 0]
            oy = origin[1] - poles[:, 1]
            a = (d[:, 0] ** 2 + d[:, 1] ** 2)[:, None]
            b = 2.0 * (d[:, 0:1] * ox[None, :] + d[:, 1:2] * oy[None, :])
            c = (ox ** 2 + oy ** 2 - self.pole_radius ** 2)[None, :]
            disc = b * b - 4.0 * a * c
            with np.errstate(divide="ignore", invalid="ignore"):
                tp = (-b - np.sqrt(np.where(disc >= 0, disc, np.nan))) / (2.0 * a)
            z = origin[2] + tp * d[:, 2:3]
            okp = (disc >= 0) & (tp > 1e-6) & (z >= 0.0) & (z <= self.pole_height)
            tp = np.where(okp, tp, np.inf)
            t = np.minimum(t, tp.min(axis=1))
            out[s:s + chunk] = t
        return out

    def lidar_scan(self, T_sensor, rng, rings=64, azimuths=2048, elev_deg=(2.0, -24.8),
                   max_range=100.0, range_noise=0.02, dropout=0.10):
        """One spinning-LiDAR frame; returns f32[N,3] points in the SENSOR frame."""
        el = np.radians(np.linspace(elev_deg[0], elev_deg[1], rings))
        az = np.linspace(0.0, 2.0 * math.pi, azimuths, endpoint=False)
        ee, aa = np.meshgrid(el, az, indexing="ij")
        d_s = np.stack([np.cos(ee) * np.cos(aa), np.cos(ee) * np.sin(aa), np.sin(ee)], axis=-1).reshape(-1, 3)
        R, t = T_sensor
        d_w = d_s @ R.T
        rng_t = self.raycast(t, d_w, max_range=max_range)
        keep = np.isfinite(rng_t)
        rng_t = rng_t + rng.normal(0.0, range_noise, size=rng_t.shape)
        keep &= rng_t <= max_range
        keep &= rng_t > 0.5
        keep &= rng.random(rng_t.shape) >= dropout
        pts = d_s[keep] * rng_t[keep, None]
        return pts.astype(F32)

    def _under_a_box(self, q, cell=32.0):
        """q (n,>=2): True where (x, y) lies strictly inside a box footprint.  Exact test
        |x - cx| < sx/2 and |y - cy| < sy/2 against every box, evaluated per 32 m grid cell
        against only the boxes that overlap the cell (same predicate, fewer pairs)."""
        bx = self.boxes
        half = self.extent / 2.0
        nc = int(math.ceil(self.extent / cell))
        ix = np.clip(np.floor((q[:, 0] + half) / cell).astype(np.int64), 0, nc - 1)
        iy = np.clip(np.floor((q[:, 1] + half) / cell).astype(np.int64), 0, nc - 1)
        cid = ix * nc + iy
        order = np.argsort(cid, kind="stable")
        cs = cid[order]
        starts = np.nonzero(np.r_[True, cs[1:] != cs[:-1]])[0]
        ends = np.r_[starts[1:], cs.size]
        blo = np.stack([bx[:, 0] - bx[:, 2] / 2, bx[:, 1] - bx[:, 3] / 2], axis=1)
        bhi = np.stack([bx[:, 0] + bx[:, 2] / 2, bx[:, 1] + bx[:, 3] / 2], axis=1)
        inside = np.zeros(q.shape[0], dtype=bool)
        for s, e in zip(starts, ends):
            c = int(cs[s])
            cx0 = (c // nc) * cell - half
            cy0 = (c % nc) * cell - half
            # boxes whose footprint can contain a point of this cell (clipped points sit in edge cells: pad them)
            pad = cell if (c // nc in (0, nc - 1) or c % nc in (0, nc - 1)) else 0.0
            sel = (bhi[:, 0] >= cx0 - pad) & (blo[:, 0] <= cx0 + cell + pad) & \
                  (bhi[:, 1] >= cy0 - pad) & (blo[:, 1] <= cy0 + cell + pad)
            if not sel.any():
                continue
            b = bx[sel]
            idx = order[s:e]
            pts = q[idx]
            ins = (np.abs(pts[:, None, 0] - b[None, :, 0]) < b[None, :, 2] / 2) & \
                  (np.abs(pts[:, None, 1] - b[None, :, 1]) < b[None, :, 3] / 2)
            inside[idx] = ins.any(axis=1)
        return inside

    # ---- area-uniform surface samples ------------------------------------
    def sample_surfaces(self, n, rng, center=(0.0, 0.0), radius=None, noise=0.0):
        """n area-uniform samples of the scene surfaces (ground, box walls and roofs, poles).

        With `radius`, only surfaces within that horizontal distance of `center`
        are sampled (by rejection); otherwise the whole square extent is used.
        Returns f32[n,3] in the map frame.
        """
        half = self.extent / 2.0
        bx = self.boxes
        wall_area = 2.0 * (bx[:, 2] + bx[:, 3]) * bx[:, 4]
        roof_area = bx[:, 2] * bx[:, 3]
        pole_area = np.full(len(self.poles), 2.0 * math.pi * self.pole_radius * self.pole_height)
        ground_area = self.extent ** 2
        areas = np.concatenate([[ground_area], wall_area, roof_area, pole_area])
        prob = areas / areas.sum()
        nb = len(bx)
        out = np.empty((0, 3))
        cx, cy = center
        while out.shape[0] < n:
            m = int((n - out.shape[0]) * (1.3 if radius is None else
                                          1.3 * self.extent ** 2 / (math.pi * radius ** 2))) + 1024
            m = min(m, 8_000_000)
            face = rng.choice(len(areas), size=m, p=prob)
            u = rng.random(m)
            w = rng.random(m)
            p = np.empty((m, 3))
            g = face == 0
            p[g, 0] = (u[g] * 2 - 1) * half
            p[g, 1] = (w[g] * 2 - 1) * half
            p[g, 2] = 0.0
            wl = (face >= 1) & (face <= nb)
            bi = face[wl] - 1
            sx, sy, hh = bx[bi, 2], bx[bi, 3], bx[bi, 4]
            per = u[wl] * 2.0 * (sx + sy)
            # walk the perimeter: +y side, +x side, -y side, -x side
            x = np.where(per < sx, per - sx / 2,
                np.where(per < sx + sy, sx / 2,
                np.where(per < 2 * sx + sy, sx / 2 - (per - sx - sy), -sx / 2)))
            y = np.where(per < sx, sy / 2,
                np.where(per < sx + sy, sy / 2 - (per - sx),
                np.where(per < 2 * sx + sy, -sy / 2, -sy / 2 + (per - 2 * sx - sy))))
            p[wl, 0] = bx[bi, 0] + x
            p[wl, 1] = bx[bi, 1] + y
            p[wl, 2] = w[wl] * hh
            rf = (face > nb) & (face <= 2 * nb)
            bi = face[rf] - 1 - nb
            p[rf, 0] = bx[bi, 0] + (u[rf] - 0.5) * bx[bi, 2]
            p[rf, 1] = bx[bi, 1] + (w[rf] - 0.5) * bx[bi, 3]
            p[rf, 2] = bx[bi, 4]
            pl = face > 2 * nb
            pi = face[pl] - 1 - 2 * nb
            ang = u[pl] * 2.0 * math.pi
            p[pl, 0] = self.poles[pi, 0] + self.pole_radius * np.cos(ang)
            p[pl, 1] = self.poles[pi, 1] + self.pole_radius * np.sin(ang)
            p[pl, 2] = w[pl] * self.pole_height
            keep = np.ones(m, dtype=bool)
            if radius is not None:
                keep &= (p[:, 0] - cx) ** 2 + (p[:, 1] - cy) ** 2 <= radius ** 2
            # ground samples under a building are not visible surfaces: drop them
            gi = np.nonzero(g & keep)[0]
            if gi.size:
                keep[gi[self._under_a_box(p[gi])]] = False
            out = np.concatenate([out, p[keep]], axis=0)
        out = out[:n]
        if noise > 0:
            out = out + rng.normal(0.0, noise, size=out.shape)
        return out.astype(F32)


def c2_single_frame(seed=1, n_map_candidates=1_520_000, map_radius=150.0, rings=64, azimuths=2048,
                    scene=None, sensor_xy=(0.0, 0.0)):
    """BASELINE.json configs[1]: one 64 x 2048 frame against a ~1.5 M-point local map.

    Returns dict(scene, map_points (candidates offered to the map, f32[n,3] map frame),
    scan (raw scan, sensor frame), T_gt, T_init (0.5 m / 3 deg perturbation), voxel=1.0,
    cap=20, sigma=2.0, max_iters=30).  `n_map_candidates` is the number of area-uniform
    surface samples offered; with voxel 1.0 m and cap 20 about 1.5 M of them are stored
    (calibrated with the oracle).
    """
    rng = np.random.default_rng(seed)
    if scene is None:
        scene = UrbanScene(seed=seed)
    T_gt = pose_from_rpy_t(0.0, 0.0, math.radians(7.0), [sensor_xy[0], sensor_xy[1], 1.8])
    scan = scene.lidar_scan(T_gt, rng, rings=rings, azimuths=azimuths)
    map_pts = scene.sample_surfaces(n_map_candidates, rng, center=sensor_xy, radius=map_radius)
    T_init = perturb_pose(T_gt, 0.5, 3.0, rng)
    return dict(scene=scene, map_points=map_pts, scan=scan, T_gt=T_gt, T_init=T_init,
                voxel=1.0, cap=20, sigma=2.0, max_iters=30)


# --------------------------------------------------------------------------
# C3: racing sequence -- straight + constant-radius arc, analytic surfaces
# --------------------------------------------------------------------------
@dataclass
class RaceTrack:
    seed: int = 2
    straight: float = 1000.0     # [m] along +x from x=0
    radius: float = 500.0        # left-hand arc after the straight
    arc_length: float = 1000.0
    half_width: float = 8.0
    wall_height: float = 1.2
    pole_spacing: float = 50.0
    pole_offset: float = 9.0
    pole_radius: float = 0.15
    pole_height: float = 8.0
    poles: np.ndarray = field(init=False)

    def __post_init__(self):
        s = np.arange(0.0, self.straight + self.arc_length + 1e-9, self.pole_spacing)
        pts = []
        for si in s:
            c, yaw = self.centerline(si)
            nrm = np.array([-math.sin(yaw), math.cos(yaw)])
            pts.append(c + self.pole_offset * nrm)
            pts.append(c - self.pole_offset * nrm)
        self.poles = np.array(pts)

    def centerline(self, s):
        """Position (x,y) and heading at arc length s."""
        if s <= self.straight:
            return np.array([s, 0.0]), 0.0
        a = (s - self.straight) / self.radius
        c = np.array([self.straight, self.radius])
        return c + self.radius * np.array([math.sin(a), -math.cos(a)]), a

    def pose_at(self, s, height=0.0):
        c, yaw = self.centerline(s)
        return pose_from_rpy_t(0.0, 0.0, yaw, [c[0], c[1], height])

    def raycast(self, origin, dirs):
        o = np.asarray(origin, dtype=np.float64)
        d = np.asarray(dirs, dtype=np.float64)
        n = d.shape[0]
        t = np.full(n, np.inf)
        amax = self.arc_length / self.radius
        cx, cy = self.straight, self.radius

        def on_track_xy(x, y, tol):
            """Is (x,y) laterally within tol of the centreline (either section)?"""
            st = (x >= 0.0) & (x <= self.straight) & (np.abs(y) <= tol)
            r = np.hypot(x - cx, y - cy)
            ang = np.arctan2(x - cx, -(y - cy))
            ar = (ang >= 0.0) & (ang <= amax) & (np.abs(r - self.radius) <= tol)
            return st | ar

        with np.errstate(divide="ignore", invalid="ignore"):
            # asphalt
            tg = -o[2] / d[:, 2]
            ok = tg > 1e-6
            xg = o[0] + tg * d[:, 0]
            yg = o[1] + tg * d[:, 1]
            ok &= on_track_xy(xg, yg, self.half_width)
            t = np.minimum(t, np.where(ok, tg, np.inf))
            # straight walls y = +-hw
            for yw in (-self.half_width, self.half_width):
                tw = (yw - o[1]) / d[:, 1]
                xw = o[0] + tw * d[:, 0]
                zw = o[2] + tw * d[:, 2]
                ok = (tw > 1e-6) & (xw >= 0.0) & (xw <= self.straight) & (zw >= 0.0) & (zw <= self.wall_height)
                t = np.minimum(t, np.where(ok, tw, np.inf))
            # arc walls: vertical cylinders radius R -+ hw about (cx, cy); both roots
            ox, oy = o[0] - cx, o[1] - cy
            a = d[:, 0] ** 2 + d[:, 1] ** 2
            b = 2.0 * (d[:, 0] * ox + d[:, 1] * oy)
            for rw in (self.radius - self.half_width, self.radius + self.half_width):
                c = ox * ox + oy * oy - rw * rw
                disc = b * b - 4 * a * c
                sq = np.sqrt(np.where(disc >= 0, disc, np.nan))
                for sign in (-1.0, 1.0):
                    tw = (-b + sign * sq) / (2 * a)
                    xw = o[0] + tw * d[:, 0]
                    yw = o[1] + tw * d[:, 1]
                    zw = o[2] + tw * d[:, 2]
                    ang = np.arctan2(xw - cx, -(yw - cy))
                    ok = (disc >= 0) & (tw > 1e-6) & (ang >= 0) & (ang <= amax) & (zw >= 0) & (zw <= self.wall_height)
                    t = np.minimum(t, np.where(ok, tw, np.inf))
            # poles
            pox = o[0] - self.poles[:, 0]
            poy = o[1] - self.poles[:, 1]
            near = np.hypot(pox, poy) < 260.0
            for px, py in zip(pox[near], poy[near]):
                bb = 2.0 * (d[:, 0] * px + d[:, 1] * py)
                cc = px * px + py * py - self.pole_radius ** 2
                disc = bb * bb - 4 * a * cc
                tp = (-bb - np.sqrt(np.where(disc >= 0, disc, np.nan))) / (2 * a)
                zp = o[2] + tp * d[:, 2]
                ok = (disc >= 0) & (tp > 1e-6) & (zp >= 0) & (zp <= self.pole_height)
                t = np.minimum(t, np.where(ok, tp, np.inf))
        return t


def c3_racing_frame(track, s, rng, rows=200, cols=300, yaw_deg=(-50.0, 0.0, 50.0), hfov_deg=120.0,
                    elev_deg=(5.0, -20.0), sensor_height=1.0, max_range=200.0, range_noise=0.02,
                    dropout=0.10):
    """One concatenated frame of three forward LiDARs at arc length s.

    Returns (scan f32[N,3] in the vehicle/sensor frame, T_gt map_from_sensor)."""
    T = track.pose_at(s, sensor_height)
    el = np.radians(np.linspace(elev_deg[0], elev_deg[1], rows))
    parts = []
    for yd in yaw_deg:
        az = np.radians(yd + np.linspace(-hfov_deg / 2, hfov_deg / 2, cols))
        ee, aa = np.meshgrid(el, az, indexing="ij")
        parts.append(np.stack([np.cos(ee) * np.cos(aa), np.cos(ee) * np.sin(aa), np.sin(ee)], axis=-1).reshape(-1, 3))
    d_s = np.concatenate(parts, axis=0)
    d_w = d_s @ T[0].T
    r = track.raycast(T[1], d_w)
    keep = np.isfinite(r)
    r = r + rng.normal(0.0, range_noise, size=r.shape)
    keep &= (r <= max_range) & (r > 0.5)
    keep &= rng.random(r.shape) >= dropout
    return (d_s[keep] * r[keep, None]).astype(F32), T


# --------------------------------------------------------------------------
# C4: map-insert stress
# --------------------------------------------------------------------------
def c4_insert_stress(seed=3, n_uniform=8_000_000, n_clustered=2_000_000, n_patches=50):
    """BASELINE.json configs[3]: uniform volume points + 20 % on random planar patches, shuffled."""
    rng = np.random.default_rng(seed)
    uni = np.empty((n_uniform, 3), dtype=F32)
    uni[:, 0] = rng.uniform(-200.0, 200.0, size=n_uniform)
    uni[:, 1] = rng.uniform(-200.0, 200.0, size=n_uniform)
    uni[:, 2] = rng.uniform(0.0, 20.0, size=n_uniform)
    per = n_clustered // n_patches
    cl = []
    for _ in range(n_patches):
        c = np.array([rng.uniform(-180, 180), rng.uniform(-180, 180), rng.uniform(2, 18)])
        nrm = rng.normal(size=3)
        nrm /= np.linalg.norm(nrm)
        e1 = np.cross(nrm, [0.0, 0.0, 1.0] if abs(nrm[2]) < 0.9 else [1.0, 0.0, 0.0])
        e1 /= np.linalg.norm(e1)
        e2 = np.cross(nrm, e1)
        uv = rng.uniform(-20.0, 20.0, size=(per, 2))
        off = rng.normal(0.0, 0.02, size=per)
        cl.append((c + uv[:, 0:1] * e1 + uv[:, 1:2] * e2 + off[:, None] * nrm).astype(F32))
    allp = np.concatenate([uni] + cl, axis=0)
    perm = rng.permutation(allp.shape[0])
    return allp[perm]


# --------------------------------------------------------------------------
# C5: NN-query sweep
# --------------------------------------------------------------------------
def c5_nn_sweep(seed=4, n_map=20_000_000, n_query=1_000_000, extent=1000.0):
    """BASELINE.json configs[4]: map samples of a 1 x 1 km urban scene and 1 M queries.

    Queries: first half = map points + N(0, 0.1 m) (hit path), second half uniform in the
    bounding box (mostly miss path); `order` is a random permutation to apply for the
    mixed run.  Returns dict(map_points, queries, is_hit, order, morton_order)."""
    rng = np.random.default_rng(seed)
    scale = (extent / 400.0) ** 2
    scene = UrbanScene(seed=seed, extent=extent, n_boxes=int(300 * scale), n_poles=int(200 * scale))
    parts = []
    left = n_map
    while left > 0:
        m = min(left, 4_000_000)
        parts.append(scene.sample_surfaces(m, rng, noise=0.02))
        left -= m
    map_pts = np.concatenate(parts, axis=0)
    nh = n_query // 2
    sel = rng.integers(0, n_map, size=nh)
    hit = (map_pts[sel].astype(np.float64) + rng.normal(0.0, 0.1, size=(nh, 3))).astype(F32)
    lo = map_pts.min(axis=0).astype(np.float64)
    hi = map_pts.max(axis=0).astype(np.float64)
    miss = rng.uniform(lo, hi, size=(n_query - nh, 3)).astype(F32)
    q = np.concatenate([hit, miss], axis=0)
    is_hit = np.concatenate([np.ones(nh, bool), np.zeros(n_query - nh, bool)])
    order = rng.permutation(n_query)
    # Morton order of the queries on a 1 m grid (an ordering of the inputs only)
    g = np.clip(((q.astype(np.float64) - lo) / 1.0).astype(np.int64), 0, (1 << 20) - 1)

    def spread(v):
        v = v & 0x1FFFFF
        v = (v | (v << 32)) & 0x1F00000000FFFF
        v = (v | (v << 16)) & 0x1F0000FF0000FF
        v = (v | (v << 8)) & 0x100F00F00F00F00F
        v = (v | (v << 4)) & 0x10C30C30C30C30C3
        v = (v | (v << 2)) & 0x1249249249249249
        return v
    code = spread(g[:, 0]) | (spread(g[:, 1]) << 1) | (spread(g[:, 2]) << 2)
    morton = np.argsort(code, kind="stable")
    return dict(map_points=map_pts, queries=q, is_hit=is_hit, order=order, morton_order=morton)


# --------------------------------------------------------------------------
# a scan distorted by ego motion during the sweep
# --------------------------------------------------------------------------
def _twist_matrix(xi):
    """4x4 matrix of the body twist xi = (v, w)"""
    v, w = xi[:3], xi[3:]
    return np.array([[0.0, -w[2], w[1], v[0]],
                     [w[2], 0.0, -w[0], v[1]],
                     [-w[1], w[0], 0.0, v[2]],
                     [0.0, 0.0, 0.0, 0.0]])


def motion_distorted_scan(seed=5, n=20000, duration=0.1, steps=1000, a=None, b=None, scene_radius=60.0,
                          history=12, history_span=0.2, history_noise=0.0):
    """Forward model of a sweep taken while the sensor moves (the INPUT of motion undistortion; none of the
    method's arithmetic): static world points W, given in the sensor frame at the frame reference time t_ref (the
    time of the last point), are observed one after the other while the sensor follows the body twist
    xi(t) = a + b (t - t_ref).  The sensor pose relative to the t_ref pose, G(t), solves dG/dt = G [xi(t)]^ with
    G(t_ref) = I; it is integrated backwards on a grid of `steps` intervals with scipy's matrix exponential at the
    interval midpoints (error O(dt^3) per step, far below fp32 resolution) and the point times are grid times, so
    `observed` is exact to integration error:  observed_i = fl32(G(t_i)^-1 W_i).

    Returns dict(observed f32[n,3], time f32[n] (offset from the first point), dt_ref, world f64[n,3], a, b,
    hist_times f64[history], hist_vel f64[history,6]) -- the history samples the twist line (+ optional noise)
    over the `history_span` seconds before t_ref, in absolute time with t_ref = 100.0 s."""
    from scipy.linalg import expm

    rng = np.random.default_rng(seed)
    if a is None:
        a = np.array([69.4, 0.3, -0.1, 0.01, -0.02, 0.25])     # ~250 km/h forward, gentle yaw rate
    if b is None:
        b = np.array([-4.0, 0.5, 0.0, 0.0, 0.0, 0.6])
    a, b = np.asarray(a, dtype=np.float64), np.asarray(b, dtype=np.float64)
    dt = duration / steps
    # G at grid times t_ref - j dt, j = 0..steps (backwards): G(t - dt) = G(t) expm(-[xi(t - dt/2)]^ dt)
    G = np.empty((steps + 1, 4, 4))
    G[0] = np.eye(4)
    for j in range(steps):
        tm = -(j + 0.5) * dt                                    # midpoint, relative to t_ref
        G[j + 1] = G[j] @ expm(-_twist_matrix(a + b * tm) * dt)
    # spinning-LiDAR-like ordering: the point's time grows with its azimuth
    az = np.sort(rng.uniform(-math.pi, math.pi, n))
    rad = rng.uniform(2.0, scene_radius, n)
    z = rng.uniform(-2.0, 8.0, n)
    world = np.stack([rad * np.cos(az), rad * np.sin(az), z], axis=1)
    grid = np.minimum((np.arange(n) * (steps + 1)) // n, steps)    # 0 = first point ... steps = last point (t_ref)
    back = steps - grid                                            # number of intervals before t_ref
    Gi = np.linalg.inv(G[back])                                    # (n,4,4)
    obs = np.einsum("nij,nj->ni", Gi[:, :3, :3], world) + Gi[:, :3, 3]
    time = (grid * dt).astype(F32)
    t_ref = 100.0
    ht = t_ref - history_span + history_span * (np.arange(history) + 0.5) / history
    hv = a[None, :] + b[None, :] * (ht - t_ref)[:, None] + rng.normal(0.0, history_noise, (history, 6))
    return dict(observed=obs.astype(F32), time=time, dt_ref=float(duration), world=world, a=a, b=b,
                hist_times=ht, hist_vel=hv, t_ref=t_ref)
