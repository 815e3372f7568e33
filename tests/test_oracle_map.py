"""Pins for the oracle's voxel key, voxelise, capped insert, prune and 27-voxel NN (A1-A6).

Each test checks oracle/ against something other than itself: hand-evaluated fixtures under
tests/golden/, NumPy/SciPy library routines, closed forms, brute force, or invariants.
"""
import numpy as np
import pytest
from scipy.spatial import cKDTree

import far_scenes as fs
import oracle
from helpers import (export_to_dict, load_golden, np_capped_contents, np_nn_bruteforce, np_pack, np_unpack,
                     np_voxel_index)


# ----------------------------------------------------------------------------- A1 keys
def test_key_floor_golden():
    g = load_golden("key_examples.json")
    for x, want in g["floor_cases"]:
        k, valid = oracle.keys(np.array([[x, 0.0, 0.0]], dtype=np.float32), g["voxel"])
        assert valid[0]
        assert oracle.unpack_key(k[0])[0] == want, (x, want)


def test_key_pack_golden_and_roundtrip():
    g = load_golden("key_examples.json")
    for k3, hx in g["pack_cases"]:
        assert oracle.pack_key(*k3) == int(hx, 16)
        assert oracle.unpack_key(int(hx, 16)).tolist() == k3
    rng = np.random.default_rng(0)
    for k3 in rng.integers(-(1 << 20), 1 << 20, size=(200, 3)):
        key = oracle.pack_key(*k3)
        assert key >> 63 == 0                      # bit 63 is free: sentinels cannot collide
        assert oracle.unpack_key(key).tolist() == k3.tolist()
        assert key == int(np_pack(k3[None])[0])


@pytest.mark.parametrize("voxel", [0.25, 0.5, 1.0, 2.0, 4.0, 0.3])
def test_key_matches_numpy_floor(voxel):
    rng = np.random.default_rng(1)
    pts = (rng.normal(size=(20000, 3)) * 50).astype(np.float32)
    # exact multiples of the voxel size sit on boundaries: include them
    pts[:2000] = (rng.integers(-300, 300, size=(2000, 3)) * voxel).astype(np.float32)
    k, valid = oracle.keys(pts, voxel)
    assert valid.all()
    want = np_voxel_index(pts, voxel)
    assert np.array_equal(np_unpack(k), want)
    assert np.array_equal(k, np_pack(want))


def test_key_invalid_points():
    pts = np.array([[np.nan, 0, 0], [0, np.inf, 0], [0, 0, -np.inf], [1e7, 0, 0], [-1e7, 0, 0],
                    [524287.9, 0, 0], [524288.0, 0, 0], [-524288.0, 0, 0], [-524288.1, 0, 0]], dtype=np.float32)
    _, valid = oracle.keys(pts, 0.5)      # index range is [-2^20, 2^20) -> |x| < 524288 m at v = 0.5
    assert valid.tolist() == [False, False, False, False, False, True, False, True, False]


# ----------------------------------------------------------------------------- A2 voxelise
def _scan(seed=5, n=30000):
    rng = np.random.default_rng(seed)
    return (rng.normal(size=(n, 3)) * [20, 20, 2]).astype(np.float32)


@pytest.mark.parametrize("voxel", [0.5, 1.0])
def test_voxelize_matches_numpy_unique(voxel):
    pts = _scan()
    out, idx = oracle.voxelize(pts, voxel)
    keys = np_pack(np_voxel_index(pts, voxel))
    _, first = np.unique(keys, return_index=True)
    assert len(idx) == len(first)
    assert np.array_equal(idx, np.sort(first))            # ascending source index
    assert np.array_equal(out, pts[idx])                   # outputs are a subset of the inputs, bit-exact


def test_voxelize_idempotent_and_reverse():
    pts = _scan(6, 5000)
    out, idx = oracle.voxelize(pts, 1.0)
    out2, idx2 = oracle.voxelize(out, 1.0)
    assert np.array_equal(out2, out) and np.array_equal(idx2, np.arange(len(out)))
    # reversing the input makes the former LAST point of each voxel the representative
    rev = pts[::-1].copy()
    _, idxr = oracle.voxelize(rev, 1.0)
    keys = np_pack(np_voxel_index(pts, 1.0))
    last = {}
    for i, k in enumerate(keys):
        last[int(k)] = i
    assert sorted(len(pts) - 1 - idxr) == sorted(last.values())


def test_voxelize_skips_invalid():
    pts = np.array([[0.1, 0.1, 0.1], [np.nan, 0, 0], [0.2, 0.1, 0.1], [5, 5, 5]], dtype=np.float32)
    out, idx = oracle.voxelize(pts, 0.5)
    assert idx.tolist() == [0, 3]


# ----------------------------------------------------------------------------- A3/A4 insert
def test_insert_golden_example():
    g = load_golden("insert_worked_example.json")
    m = oracle.Map(g["voxel"], g["cap"])
    st = m.insert(np.array(g["points"], dtype=np.float32))
    d = export_to_dict(m.export())
    want = {oracle.pack_key(*map(int, k.split(","))): v for k, v in g["expect"].items()}
    assert {k: [e[0] for e in v] for k, v in d.items()} == want
    assert st["n_accepted"] == 3 and st["n_new_voxels"] == 2 and st["n_offered"] == 4


@pytest.mark.parametrize("cap", [1, 4, 20])
def test_insert_contents_match_stable_argsort(cap):
    rng = np.random.default_rng(2)
    pts = (rng.normal(size=(20000, 3)) * [3, 3, 0.5]).astype(np.float32)
    m = oracle.Map(0.5, cap)
    st = m.insert(pts)
    exp = m.export()
    got = {k: [e[0] for e in v] for k, v in export_to_dict(exp).items()}
    want = np_capped_contents(pts, 0.5, cap)
    assert got == want
    keys = np_pack(np_voxel_index(pts, 0.5))
    _, mult = np.unique(keys, return_counts=True)
    assert np.array_equal(exp["counts"], np.minimum(mult, cap))     # export is sorted by key, like np.unique
    assert exp["counts"].max() <= cap
    assert st["n_accepted"] == exp["counts"].sum()
    # stored coordinates are the offered fp32 bits
    for v in range(0, len(exp["keys"]), 97):
        for j in range(exp["counts"][v]):
            assert np.array_equal(exp["xyz"][v, j], pts[exp["ids"][v, j]])
    # ids strictly increasing inside a voxel
    for v in range(len(exp["keys"])):
        ids = exp["ids"][v, :exp["counts"][v]].astype(np.int64)
        assert np.all(np.diff(ids) > 0)


def test_insert_batch_invariance():
    rng = np.random.default_rng(3)
    pts = (rng.normal(size=(12000, 3)) * [4, 4, 1]).astype(np.float32)
    a = oracle.Map(0.5, 5)
    a.insert(pts)
    b = oracle.Map(0.5, 5)
    for s in range(0, len(pts), 1000):
        b.insert(pts[s:s + 1000])
    assert export_to_dict(a.export()) == export_to_dict(b.export())
    assert a.size() == b.size() and a.size()[2] == len(pts)


def test_insert_with_pose_matches_float64_transform():
    rng = np.random.default_rng(4)
    pts = (rng.normal(size=(3000, 3)) * 10).astype(np.float32)
    T = fs.pose_from_rpy_t(0.1, -0.2, 0.7, [3.0, -2.0, 0.5])
    m = oracle.Map(1.0, 50)
    m.insert(pts, pose=T)
    exp = m.export()
    R, t = T
    p64 = pts.astype(np.float64)
    want = np.empty_like(p64)
    for r in range(3):       # ((R0*x + R1*y) + R2*z) + t, each op rounded in binary64
        want[:, r] = ((R[r, 0] * p64[:, 0] + R[r, 1] * p64[:, 1]) + R[r, 2] * p64[:, 2]) + t[r]
    want = want.astype(np.float32)
    for v in range(len(exp["keys"])):
        for j in range(exp["counts"][v]):
            assert np.array_equal(exp["xyz"][v, j], want[exp["ids"][v, j]])


def test_insert_invalid_points_consume_ids():
    pts = np.array([[0.1, 0.1, 0.1], [np.nan, 0, 0], [0.2, 0.1, 0.1]], dtype=np.float32)
    m = oracle.Map(0.5, 4)
    st = m.insert(pts)
    assert st["n_invalid"] == 1 and st["n_accepted"] == 2
    d = export_to_dict(m.export())
    assert [e[0] for e in d[oracle.pack_key(0, 0, 0)]] == [0, 2]
    assert m.size()[2] == 3


# ----------------------------------------------------------------------------- A5 prune
def test_prune_closed_form_and_noop():
    rng = np.random.default_rng(7)
    pts = (rng.uniform(-30, 30, size=(20000, 3))).astype(np.float32)
    m = oracle.Map(1.0, 3)
    m.insert(pts)
    before = m.export()
    st0 = m.prune([0, 0, 0], np.inf)
    assert st0["n_voxels_removed"] == 0 and export_to_dict(m.export()) == export_to_dict(before)
    c = np.array([1.5, -2.25, 0.75])
    r = 17.0
    st = m.prune(c, r)
    after = m.export()
    k = np_unpack(before["keys"]).astype(np.float64)
    d = (k + 0.5) * 1.0 - c
    d2 = (d[:, 0] * d[:, 0] + d[:, 1] * d[:, 1]) + d[:, 2] * d[:, 2]
    keep = ~(d2 > r * r)
    assert np.array_equal(after["keys"], before["keys"][keep])
    assert st["n_voxels_removed"] == int((~keep).sum())
    assert st["n_points_removed"] == int(before["counts"][~keep].sum())
    assert st["n_voxels_left"] == int(keep.sum())


def test_prune_then_reinsert_equals_fresh_region():
    rng = np.random.default_rng(8)
    pts = (rng.uniform(-10, 10, size=(8000, 3))).astype(np.float32)
    m = oracle.Map(1.0, 2)
    m.insert(pts)
    before = m.export()
    m.prune([0, 0, 0], 6.0)
    kept_keys = set(m.export()["keys"].tolist())
    removed_keys = set(before["keys"].tolist()) - kept_keys
    m.insert(pts)       # ids 8000.. ; removed voxels are recreated empty and refilled
    d = export_to_dict(m.export())
    fresh = np_capped_contents(pts, 1.0, 2, first_id=8000)
    for k in removed_keys:
        assert [e[0] for e in d[k]] == fresh[k]
    # NN never returns a removed id
    ids, _ = m.nn(pts[:500])
    removed_ids = {i for k in removed_keys for i in np_capped_contents(pts, 1.0, 2)[k]}
    assert not (set(ids.tolist()) & removed_ids)


# ----------------------------------------------------------------------------- A6 NN
def test_nn_golden_example():
    g = load_golden("nn_worked_example.json")
    m = oracle.Map(g["voxel"], 20)
    m.insert(np.array(g["stored"], dtype=np.float32))
    for case in g["queries"]:
        ids, d2 = m.nn(np.array([case["q"]], dtype=np.float32))
        assert ids[0] == case["id"], case
        if case["d2"] == "inf":
            assert np.isinf(d2[0])
        else:
            assert d2[0] == pytest.approx(case["d2"], rel=1e-5)
    t = g["tie"]
    m2 = oracle.Map(g["voxel"], 20)
    m2.insert(np.array(t["stored"], dtype=np.float32))
    ids, _ = m2.nn(np.array([t["q"]], dtype=np.float32))
    assert ids[0] == t["id"]


def _c1_map():
    c1 = fs.c1_tiny()
    m = oracle.Map(c1["voxel"], c1["cap"])
    m.insert(c1["map_points"])
    return c1, m


def test_nn_vs_numpy_bruteforce_c1():
    c1, m = _c1_map()
    exp = m.export()
    sel = np.concatenate([np.arange(c) + v * m.cap for v, c in enumerate(exp["counts"])])
    sx = exp["xyz"].reshape(-1, 3)[sel]
    sid = exp["ids"].reshape(-1)[sel]
    rng = np.random.default_rng(9)
    q = np.concatenate([c1["scan"][:300], rng.uniform(-6, 6, size=(200, 3)).astype(np.float32)])
    ids, d2 = m.nn(q)
    wid, wd2 = np_nn_bruteforce(sx, sid, q, c1["voxel"])
    assert np.array_equal(ids, wid)
    assert np.array_equal(d2, wd2.astype(np.float32))
    bid, bd2 = m.nn_brute(q)
    assert np.array_equal(ids, bid) and np.array_equal(d2, bd2)
    assert (ids == oracle.NO_ID).any() and (ids != oracle.NO_ID).any()


def test_nn_vs_ckdtree_when_within_voxel():
    """Any point within v of q lies in an adjacent voxel, so if d <= v the result is the global NN."""
    c1, m = _c1_map()
    exp = m.export()
    sel = np.concatenate([np.arange(c) + v * m.cap for v, c in enumerate(exp["counts"])])
    sx = exp["xyz"].reshape(-1, 3)[sel].astype(np.float64)
    sid = exp["ids"].reshape(-1)[sel]
    tree = cKDTree(sx)
    rng = np.random.default_rng(10)
    q = np.concatenate([c1["scan"], rng.uniform(-6, 6, size=(2000, 3)).astype(np.float32)])
    ids, d2 = m.nn(q)
    dist, j = tree.query(q.astype(np.float64), k=2)
    checked = 0
    for i in range(len(q)):
        if dist[i, 0] <= c1["voxel"]:
            assert ids[i] != oracle.NO_ID
            assert d2[i] == pytest.approx(dist[i, 0] ** 2, rel=1e-6, abs=1e-12)
            if dist[i, 1] > dist[i, 0] * (1 + 1e-9):       # unique minimum: the id must match too
                assert ids[i] == sid[j[i, 0]]
            checked += 1
    assert checked > 1000


def test_nn_multithreaded_equals_single():
    c1, m = _c1_map()
    a = m.nn(c1["scan"], nthreads=1)
    b = m.nn(c1["scan"], nthreads=4)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])


def test_renumber_shifts_ids_by_the_minimum_and_nothing_else():
    """R22 pin: after renumbering, the stored ids are the old ones minus their minimum (so order, contents, NN winners and
    tie-breaks are those of the old ids), the counter moves by the same amount, and later ids continue from it."""
    rng = np.random.default_rng(31)
    pts = rng.uniform(-6, 6, size=(5000, 3)).astype(np.float32)
    m = oracle.Map(1.0, 4)
    m.insert(pts)
    m.prune([20.0, 0.0, 0.0], 16.5)          # removes the voxels that hold the earliest ids near x = -6 ... some survive elsewhere
    m.insert(pts[:100] + np.float32(0.01))
    before = m.export()
    stored = before["counts"][:, None] > np.arange(4)[None, :]
    mn = int(before["ids"][stored].min())
    nid = m.size()[2]
    q = rng.uniform(-6, 6, size=(500, 3)).astype(np.float32)
    ids0, d0 = m.nn(q)
    sub = m.renumber()
    after = m.export()
    assert sub == mn and m.size()[2] == nid - mn
    assert np.array_equal(after["keys"], before["keys"]) and np.array_equal(after["counts"], before["counts"])
    assert np.array_equal(after["xyz"], before["xyz"])
    assert np.array_equal(after["ids"][stored].astype(np.int64), before["ids"][stored].astype(np.int64) - mn)
    ids1, d1 = m.nn(q)
    hit = ids0 != oracle.NO_ID
    assert np.array_equal(ids1[hit].astype(np.int64), ids0[hit].astype(np.int64) - mn) and np.array_equal(d1, d0)
    assert np.array_equal(ids1[~hit], ids0[~hit])
    assert m.renumber() == 0                  # idempotent: the minimum is now 0
    st = m.insert(pts[:7])
    e = m.export()
    assert int(e["ids"][e["counts"][:, None] > np.arange(4)[None, :]].max()) <= nid - mn + 6
    # an empty map restarts at 0
    m.prune([1000.0, 0.0, 0.0], 1.0)
    assert m.size()[0] == 0 and m.renumber() == nid - mn + 7 and m.size()[2] == 0


def test_clone_is_a_deep_independent_copy():
    """faro_map_clone (bookkeeping for bench.py --impl reference): the copy has the same contents, covariances and id
    counter; inserting into or pruning one of the two leaves the other as it was."""
    rng = np.random.default_rng(77)
    pts = rng.uniform(-6, 6, size=(5000, 3)).astype(np.float32)
    a = oracle.Map(0.5, 6)
    a.insert(pts[:3000], compute_cov=True)
    b = a.clone()
    ea, eb = a.export(with_cov=True), b.export(with_cov=True)
    assert a.size() == b.size() and (b.voxel, b.cap, b.k_cov) == (a.voxel, a.cap, a.k_cov)
    for k in ea:
        assert np.array_equal(ea[k], eb[k]), k
    assert b.insert(pts[3000:]) == oracle.Map.clone(a).insert(pts[3000:])      # the counter and the counts came along
    a.prune([0.0, 0.0, 0.0], 2.0)
    e2 = b.export(with_cov=True)
    assert b.size()[1] > a.size()[1] and len(e2["keys"]) > len(ea["keys"])
    ref = oracle.Map(0.5, 6)
    ref.insert(pts[:3000], compute_cov=True); ref.insert(pts[3000:])
    er = ref.export(with_cov=True)
    for k in er:
        assert np.array_equal(er[k], e2[k]), k
