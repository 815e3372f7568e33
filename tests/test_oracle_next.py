"""Pins for the oracle's motion undistortion (R15/R16) and Adaptive Submap Density
(R17).

Each test checks oracle/ against something other than itself: closed forms, NumPy/SciPy library routines
(polyfit, the matrix exponential on an independently integrated trajectory), brute-force restatements and invariants.
"""
import numpy as np
import pytest
from scipy.linalg import expm

import far_scenes as fs
import oracle
from helpers import np_pack, np_voxel_index, twist_matrix


# ------------------------------------------------------------------------------------------ R15: regression
def test_motion_fit_matches_polyfit():
    rng = np.random.default_rng(0)
    t_ref = 12.5
    times = t_ref - np.sort(rng.uniform(0.0, 0.3, 15))[::-1]
    vel = rng.normal(0, 1, (15, 6)) + np.array([60, 0, 0, 0, 0, 0.2])
    a, b = oracle.motion_fit(times, vel, t_ref)
    for c in range(6):
        slope, icpt = np.polyfit(times - t_ref, vel[:, c], 1)
        assert abs(b[c] - slope) < 1e-9 * max(1.0, abs(slope))
        assert abs(a[c] - icpt) < 1e-9 * max(1.0, abs(icpt))


def test_motion_fit_recovers_exact_line_and_degenerate_cases():
    t_ref = 3.0
    times = np.array([2.7, 2.8, 2.95, 3.0])
    a0 = np.array([10.0, -1.0, 0.5, 0.1, 0.0, -0.3])
    b0 = np.array([2.0, 0.0, -0.1, 0.0, 0.4, 1.0])
    vel = a0[None] + b0[None] * (times - t_ref)[:, None]
    a, b = oracle.motion_fit(times, vel, t_ref)
    assert np.allclose(a, a0, atol=1e-12) and np.allclose(b, b0, atol=1e-11)
    # one sample, or all samples at one time: no slope, a = mean
    a, b = oracle.motion_fit(times[:1], vel[:1], t_ref)
    assert np.array_equal(b, np.zeros(6)) and np.allclose(a, vel[0])
    a, b = oracle.motion_fit(np.full(3, 2.9), vel[:3], t_ref)
    assert np.array_equal(b, np.zeros(6)) and np.allclose(a, vel[:3].mean(axis=0))


# ------------------------------------------------------------------------------------------ R16: closed forms
def _cloud(n, seed):
    rng = np.random.default_rng(seed)
    p = rng.uniform(-80, 80, (n, 3)).astype(np.float32)
    t = np.sort(rng.uniform(0, 0.1, n)).astype(np.float32)
    return p, t


def test_undistort_zero_motion_is_identity():
    p, t = _cloud(1000, 1)
    out = oracle.undistort(p, t, 0.1, np.zeros(6), np.zeros(6))
    assert np.array_equal(out.view(np.uint32), p.view(np.uint32))


def test_undistort_points_at_reference_time_do_not_move():
    p, _ = _cloud(500, 2)
    t = np.full(500, 0.1, dtype=np.float32)
    out = oracle.undistort(p, t, float(np.float32(0.1)), [50, 1, 2, 0.1, 0.2, 0.3], [1, 2, 3, 4, 5, 6])
    assert np.array_equal(out.view(np.uint32), p.view(np.uint32))


def test_undistort_pure_translation_closed_form():
    # constant velocity v, no rotation: the sensor advances v*Delta between the point's time and t_ref, so the
    # point, seen from the later pose, lies at p - v*Delta
    p, t = _cloud(2000, 3)
    v = np.array([69.4, -2.0, 0.5])
    out = oracle.undistort(p, t, 0.1, np.r_[v, 0, 0, 0], np.zeros(6))
    D = 0.1 - t.astype(np.float64)
    want = p.astype(np.float64) - v[None] * D[:, None]
    assert np.abs(out - want).max() <= 1e-5          # fp32 rounding of the output (ulp(128) = 7.6e-6)
    # and with a linear acceleration: displacement = v*D - acc*D^2/2 (velocity is a + b (t - t_ref))
    acc = np.array([-8.0, 0.0, 1.0])
    out = oracle.undistort(p, t, 0.1, np.r_[v, 0, 0, 0], np.r_[acc, 0, 0, 0])
    want = p.astype(np.float64) - (v[None] * D[:, None] - acc[None] * (0.5 * D * D)[:, None])
    assert np.abs(out - want).max() <= 1e-5


def test_undistort_pure_yaw_closed_form():
    # constant yaw rate w about z: p' = Rz(-w*Delta) p
    p, t = _cloud(2000, 4)
    w = 0.8
    out = oracle.undistort(p, t, 0.1, [0, 0, 0, 0, 0, w], np.zeros(6))
    ang = -w * (0.1 - t.astype(np.float64))
    x, y = p[:, 0].astype(np.float64), p[:, 1].astype(np.float64)
    want = np.stack([np.cos(ang) * x - np.sin(ang) * y, np.sin(ang) * x + np.cos(ang) * y, p[:, 2].astype(np.float64)], axis=1)
    assert np.abs(out - want).max() <= 1e-5
    assert np.abs(out - p).max() > 1e-2               # the correction is not a no-op


def test_undistort_constant_twist_matches_matrix_exponential():
    # constant twist: exact solution G(t_i)^-1 G(t_ref) = expm([xi]^ Delta); the point moves by its inverse
    p, t = _cloud(300, 5)
    xi = np.array([40.0, 3.0, -1.0, 0.05, -0.1, 0.5])
    out = oracle.undistort(p, t, 0.1, xi, np.zeros(6))
    for i in range(0, 300, 7):
        D = 0.1 - float(t[i])
        E = expm(-twist_matrix(xi) * D)
        want = E[:3, :3] @ p[i].astype(np.float64) + E[:3, 3]
        assert np.abs(out[i] - want).max() <= 1e-5


@pytest.mark.parametrize("case", ["racing", "spinning", "aggressive"])
def test_undistort_recovers_static_world_from_moving_sweep(case):
    """End to end against an independent forward model (far_scenes.motion_distorted_scan integrates the sensor
    trajectory with SciPy's expm on a fine grid): undistorting the observed sweep with the true twist line must
    give back the static world as seen from the reference pose.  This is what pins the sign and the Delta^2/2
    and [a,b] Delta^3/12 terms: dropping the slope term moves points by up to ~0.2 m here, dropping the bracket
    term by ~3.5 mm (racing case), both far above the bound."""
    cfg = {"racing": dict(seed=5),
           "spinning": dict(seed=6, a=[12.0, 0.2, 0.0, 0.02, 0.01, 0.6], b=[1.5, 0.0, 0.0, 0.0, 0.0, -1.0]),
           "aggressive": dict(seed=7, a=[30.0, -5.0, 2.0, 0.5, -0.4, 1.5], b=[-20.0, 8.0, 3.0, 2.0, 1.0, -3.0])}[case]
    d = fs.motion_distorted_scan(n=6000, **cfg)
    out = oracle.undistort(d["observed"], d["time"], d["dt_ref"], d["a"], d["b"])
    err = np.linalg.norm(out.astype(np.float64) - d["world"], axis=1)
    raw = np.linalg.norm(d["observed"].astype(np.float64) - d["world"], axis=1)
    assert raw.max() > 0.5                                       # the sweep really is distorted
    # bound: fp32 rounding of input and output (2 ulp at 64 m = 1.5e-5) + third-order Magnus remainder
    assert err.max() <= (6e-5 if case == "aggressive" else 2e-5), err.max()
    # dropping the second-order term must be visible (it is the reading R16 takes)
    a, b = np.asarray(d["a"]), np.asarray(d["b"])
    bracket = np.r_[np.cross(a[3:], b[:3]) - np.cross(b[3:], a[:3]), np.cross(a[3:], b[3:])]
    assert np.linalg.norm(bracket) * d["dt_ref"] ** 3 / 12 > 5e-4 or case == "spinning"


def test_undistort_from_fitted_history():
    d = fs.motion_distorted_scan(n=3000, seed=8)
    a, b = oracle.motion_fit(d["hist_times"], d["hist_vel"], d["t_ref"])
    out = oracle.undistort(d["observed"], d["time"], d["dt_ref"], a, b)
    assert np.linalg.norm(out.astype(np.float64) - d["world"], axis=1).max() <= 2e-5


def test_undistort_nonfinite_points_pass_through():
    p, t = _cloud(16, 9)
    p[3, 1] = np.nan
    p[7, 0] = np.inf
    out = oracle.undistort(p, t, 0.1, [10, 0, 0, 0, 0, 1], np.zeros(6))
    assert np.array_equal(out[[3, 7]].view(np.uint32), p[[3, 7]].view(np.uint32))
    assert np.isfinite(out[[0, 1, 2, 4, 5, 6]]).all()


# ------------------------------------------------------------------------------------------ R17: ASMD
def _np_asmd_cap(k, voxel, c, n_close, d_max, k_min, cap):
    centre = (np.asarray(k, dtype=np.float64) + 0.5) * float(np.float32(voxel))
    d = np.sqrt(((centre - np.asarray(c, dtype=np.float64)) ** 2).sum())
    x = np.floor(n_close * (1.0 - d / d_max) + 0.5)
    return int(min(max(x, k_min), cap))


def test_asmd_cap_closed_form_and_monotone():
    rng = np.random.default_rng(0)
    c = np.array([3.0, -2.0, 1.0])
    for _ in range(300):
        k = rng.integers(-150, 150, 3)
        n_close = rng.uniform(0, 40)
        got = oracle.asmd_cap(k, 1.0, c, n_close, 100.0, 10, 20)
        assert got == _np_asmd_cap(k, 1.0, c, n_close, 100.0, 10, 20)
        assert 10 <= got <= 20
    # linear decay along a ray: non-increasing with range, = k_min at and beyond d_max, hits cap at the centre
    caps = [oracle.asmd_cap([i, 0, 0], 1.0, [0.5, 0.5, 0.5], 18.0, 100.0, 10, 20) for i in range(0, 140)]
    assert caps[0] == 18 and all(x >= y for x, y in zip(caps, caps[1:])) and caps[100] == 10 and caps[-1] == 10
    assert oracle.asmd_cap([0, 0, 0], 1.0, [0.5, 0.5, 0.5], 35.0, 100.0, 10, 20) == 20     # clamped to N_max
    # hand-evaluated: centre (10.5,0.5,0.5) from (0.5,0.5,0.5): d = 10, f = 0.9, 18*0.9 = 16.2 -> 16
    assert oracle.asmd_cap([10, 0, 0], 1.0, [0.5, 0.5, 0.5], 18.0, 100.0, 10, 20) == 16
    # 15 * (1 - 30/100) = 10.5 -> floor(11.0) = 11 (round half up)
    assert oracle.asmd_cap([30, 0, 0], 1.0, [0.5, 0.5, 0.5], 15.0, 100.0, 10, 20) == 11


def test_asmd_density_brute_force():
    c1 = fs.c1_tiny(seed=0)
    m = oracle.Map(0.5, 20)
    m.insert(c1["scan"])
    centre = np.array([1.0, 1.0, 0.0])
    for r in (0.3, 2.0, 4.0, 50.0):
        got, nv = m.asmd_density(centre, r)
        k = np_voxel_index(c1["scan"], 0.5)
        keys, counts = np.unique(np_pack(k), return_counts=True)
        counts = np.minimum(counts, 20)
        ku = np.array([k[np.nonzero(np_pack(k) == key)[0][0]] for key in keys])
        d2 = (((ku + 0.5) * 0.5 - centre) ** 2).sum(axis=1)
        sel = d2 <= r * r
        if sel.any():
            assert nv == int(sel.sum()) and got == counts[sel].sum() / sel.sum()
        else:
            assert nv == 0 and got == 20.0
    empty = oracle.Map(0.5, 20)
    assert empty.asmd_density(centre, 5.0) == (20.0, 0)


def _np_asmd_contents(xyz, voxel, cap, k_min, centre, n_close, d_max, pre=None):
    """sequential insert with the per-voxel limit, restated with a dict (ids ascending)"""
    out = {} if pre is None else {k: list(v) for k, v in pre.items()}
    ks = np_voxel_index(xyz, voxel)
    keys = np_pack(ks)
    lims = {}
    for i in range(len(xyz)):
        key = int(keys[i])
        if key not in lims:
            lims[key] = _np_asmd_cap(ks[i], voxel, centre, n_close, d_max, k_min, cap)
        lst = out.setdefault(key, [])
        if len(lst) < lims[key]:
            lst.append(i)
    return out


def test_asmd_insert_matches_brute_force_and_limits():
    rng = np.random.default_rng(3)
    # dense planar cloud out to 60 m so that both the cap and the decayed limit bind
    xy = rng.uniform(-60, 60, (300000, 2))
    pts = np.c_[xy, 0.5 + rng.normal(0, 0.02, 300000)].astype(np.float32)
    m = oracle.Map(1.0, 20)
    st = m.insert_asmd(pts, n_close=16.0, d_max=80.0)
    want = _np_asmd_contents(pts, 1.0, 20, 10, np.zeros(3), 16.0, 80.0)
    e = m.export()
    got = {int(k): [int(i) for i in e["ids"][v, :e["counts"][v]]] for v, k in enumerate(e["keys"])}
    assert got == {k: v for k, v in want.items() if v}
    assert st["n_accepted"] == sum(len(v) for v in want.values())
    # every voxel respects ITS limit; limits decay with range
    ks = {int(k): kk for k, kk in zip(np_pack(np_voxel_index(pts, 1.0)), np_voxel_index(pts, 1.0))}
    lims = {k: _np_asmd_cap(ks[k], 1.0, np.zeros(3), 16.0, 80.0, 10, 20) for k in got}
    assert all(len(got[k]) <= lims[k] for k in got)
    assert min(lims.values()) == 10 and max(lims.values()) == 16
    near = [len(v) for k, v in got.items() if np.linalg.norm(ks[k] + 0.5) < 10]
    far = [len(v) for k, v in got.items() if np.linalg.norm(ks[k] + 0.5) > 50]
    assert np.mean(near) > np.mean(far)


def test_asmd_insert_special_cases_reduce_to_plain_insert():
    c1 = fs.c1_tiny(seed=0)
    pts = c1["map_points"]
    plain = oracle.Map(0.5, 20); plain.insert(pts)
    # n_close >= cap and no decay inside the scene (d_max huge) -> the fixed cap
    a = oracle.Map(0.5, 20); a.insert_asmd(pts, n_close=40.0, d_max=1e9)
    ea, ep = a.export(), plain.export()
    assert np.array_equal(ea["keys"], ep["keys"]) and np.array_equal(ea["ids"], ep["ids"])
    # n_close = 0 -> the lower bound k everywhere = a map with cap k
    capk = oracle.Map(0.5, 10); capk.insert(pts)
    b = oracle.Map(0.5, 20); b.insert_asmd(pts, n_close=0.0, d_max=50.0)
    eb, ek = b.export(), capk.export()
    assert np.array_equal(eb["keys"], ek["keys"]) and np.array_equal(eb["counts"], ek["counts"])
    assert np.array_equal(eb["ids"][:, :10], ek["ids"])


def test_asmd_insert_with_pose_uses_pose_translation_as_centre_and_keeps_existing_points():
    rng = np.random.default_rng(4)
    pts = np.c_[rng.uniform(-30, 30, (80000, 2)), 0.5 + rng.normal(0, 0.02, 80000)].astype(np.float32)
    T = fs.pose_from_rpy_t(0.0, 0.0, 0.3, [40.0, -10.0, 0.5])
    world = fs.pose_apply(T, pts)
    m = oracle.Map(1.0, 20)
    m.insert_asmd(pts, n_close=18.0, d_max=40.0, pose=T)
    want = _np_asmd_contents(world, 1.0, 20, 10, np.asarray(T[1]), 18.0, 40.0)
    e = m.export()
    got = {int(k): [int(i) for i in e["ids"][v, :e["counts"][v]]] for v, k in enumerate(e["keys"])}
    assert got == {k: v for k, v in want.items() if v}
    # second insert from a pose 25 m further on: voxels now far from the sensor are over their new limit and take
    # nothing more, but lose nothing either (PAPER.md:109 only gates additions)
    T2 = fs.pose_from_rpy_t(0.0, 0.0, 0.3, [65.0, -10.0, 0.5])
    before = {k: list(v) for k, v in got.items()}
    m.insert_asmd(pts, n_close=18.0, d_max=40.0, pose=T2)
    e2 = m.export()
    got2 = {int(k): [int(i) for i in e2["ids"][v, :e2["counts"][v]]] for v, k in enumerate(e2["keys"])}
    for k, v in before.items():
        assert got2[k][:len(v)] == v


# ---- R21: regular spacing ("regularly spaced, with a minimum point-to-point distance of ~65 cm") -------------
def _spaced_restatement(xyz, voxel, cap, s):
    """the sequential rule written out with a dict and NumPy float64: {key: [ids]}"""
    from helpers import np_pack, np_voxel_index
    keys = np_pack(np_voxel_index(xyz, voxel))
    P = np.asarray(xyz, dtype=np.float64)
    out = {}
    for i, k in enumerate(keys.tolist()):
        ids = out.setdefault(k, [])
        if len(ids) >= cap:
            continue
        if ids:
            d = P[i] - P[ids]
            d2 = (d[:, 0] * d[:, 0] + d[:, 1] * d[:, 1]) + d[:, 2] * d[:, 2]
            if (d2 < s * s).any():
                continue
        ids.append(i)
    return out


def test_min_spacing_hand_example():
    """v = 4, s = 1: (0.5,0.5,0.5) stored; (1.0,0.5,0.5) is 0.5 away -> dropped; (1.5,0.5,0.5) is exactly 1.0 away -> stored
    (strict <); (1.9,0.5,0.5) is 0.4 from the third -> dropped; (4.1,0.5,0.5) lies 2.6 from the third but in the NEXT voxel,
    where nothing is stored -> stored; (4.3,0.5,0.5) is 0.2 from it -> dropped.  Ids are consumed by dropped points."""
    pts = np.array([[0.5, 0.5, 0.5], [1.0, 0.5, 0.5], [1.5, 0.5, 0.5], [1.9, 0.5, 0.5], [4.1, 0.5, 0.5], [4.3, 0.5, 0.5],
                    [3.9, 0.5, 0.5]], dtype=np.float32)
    m = oracle.Map(4.0, 40, min_spacing=1.0)
    st = m.insert(pts)
    e = m.export()
    stored = {int(k): [int(i) for i in ids[:c]] for k, c, ids in zip(e["keys"], e["counts"], e["ids"])}
    assert stored == {oracle.pack_key(0, 0, 0): [0, 2, 6], oracle.pack_key(1, 0, 0): [4]}     # 3.9 is 0.2 from 4.1 but in the other voxel
    assert st["n_accepted"] == 4 and st["n_new_voxels"] == 2 and m.size()[2] == 7


def test_min_spacing_matches_sequential_restatement_and_invariants():
    rng = np.random.default_rng(41)
    pts = np.concatenate([rng.uniform(-8, 8, size=(3000, 3)), rng.normal(0, 0.3, size=(3000, 3)) + [2.0, 2.0, 2.0]]).astype(np.float32)
    rng.shuffle(pts)
    v, cap, s = 4.0, 40, 4.0 / np.sqrt(40.0)                     # the paper's parameters: s = v / sqrt(N_max) = 0.632 m
    m = oracle.Map(v, cap, min_spacing=s)
    st = m.insert(pts[:3500])
    st2 = m.insert(pts[3500:])                                   # a second batch tests against what the first stored
    e = m.export()
    want = _spaced_restatement(pts, v, cap, s)
    got = {int(k): [int(i) for i in ids[:c]] for k, c, ids in zip(e["keys"], e["counts"], e["ids"])}
    assert got == want
    assert st["n_accepted"] + st2["n_accepted"] == sum(len(x) for x in want.values())
    # invariant: no two stored points of a voxel closer than s; the cap is never exceeded; ids ascend
    for v_i in range(len(e["keys"])):
        c = int(e["counts"][v_i])
        assert c <= cap
        P = e["xyz"][v_i, :c].astype(np.float64)
        if c > 1:
            d = np.linalg.norm(P[:, None, :] - P[None, :, :], axis=2) + np.eye(c) * 1e9
            assert d.min() >= s * (1 - 1e-12)
        assert (np.diff(e["ids"][v_i, :c].astype(np.int64)) > 0).all()
    # the clump at (2,2,2) would fill its voxel with near-duplicates without the rule
    plain = oracle.Map(v, cap)
    plain.insert(pts)
    assert plain.size()[1] > m.size()[1]


def test_min_spacing_zero_is_the_plain_insert():
    rng = np.random.default_rng(42)
    pts = rng.uniform(-5, 5, size=(4000, 3)).astype(np.float32)
    a, b = oracle.Map(1.0, 6), oracle.Map(1.0, 6, min_spacing=0.0)
    assert a.insert(pts) == b.insert(pts)
    ea, eb = a.export(), b.export()
    assert np.array_equal(ea["keys"], eb["keys"]) and np.array_equal(ea["ids"], eb["ids"])


def test_min_spacing_turns_ring_clumps_into_surface_patches():
    """Why PAPER.md:68 wants "regularly spaced" points.  A spinning LiDAR crosses a 4 m ground voxel with a few rings of
    densely sampled points; with the plain cap (lowest ids win) the 40 slots fill with consecutive points of the first one
    or two rings, so the k = 10 neighbourhood of a stored point is a piece of a LINE and Eq. 1's covariance has one large
    and two small eigenvalues -- its "normal" is arbitrary in the plane across the ring.  With s = v / sqrt(N_max) the
    stored points spread over the voxel and the neighbourhoods become surface patches: two comparable eigenvalues, the
    smallest eigenvector along the true normal (0, 0, 1)."""
    rng = np.random.default_rng(5)
    h = 1.8                                                          # sensor height over the plane z = 0
    elev = np.radians(np.linspace(-24.8, -3.0, 40))                  # rings that reach the ground within ~35 m
    az = np.radians(np.arange(0.0, 360.0, 360.0 / 2048))
    rings = []
    for e in elev:                                                   # ring-major order, as the sensor delivers it
        r = h / np.tan(-e)
        rings.append(np.stack([r * np.cos(az), r * np.sin(az), np.zeros_like(az)], axis=1))
    pts = (np.concatenate(rings) + rng.normal(0, 0.01, (len(elev) * len(az), 3))).astype(np.float32)
    v, cap = 4.0, 40
    quality = {}
    for name, s in (("plain", 0.0), ("spaced", v / np.sqrt(cap))):
        m = oracle.Map(v, cap, min_spacing=s)
        m.insert(pts, compute_cov=True)
        e = m.export(with_cov=True)
        ok = e["cov_valid"].astype(bool)
        C = e["cov"][ok].astype(np.float64)                          # (xx, xy, xz, yy, yz, zz)
        S = np.stack([C[:, [0, 1, 2]], C[:, [1, 3, 4]], C[:, [2, 4, 5]]], axis=1)
        w, V = np.linalg.eigh(S)                                     # ascending eigenvalues
        planarity = w[:, 1] / w[:, 2]                                # ~0 on a line, ~1 on an isotropic patch
        tilt = np.degrees(np.arccos(np.clip(np.abs(V[:, 2, 0]), 0, 1)))   # angle of the smallest eigenvector to z
        quality[name] = (float(np.median(planarity)), float(np.median(tilt)), int(ok.sum()))
    (p0, t0, n0), (p1, t1, n1) = quality["plain"], quality["spaced"]
    assert n0 > 1000 and n1 > 1000
    assert p0 < 0.05 and p1 > 5 * p0          # line-like without the rule, patches with it
    assert t1 < 2.0 and t1 < t0               # and the normals point up
