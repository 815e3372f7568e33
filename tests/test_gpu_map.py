"""GPU parity: voxel keys, voxelise, capped insert, prune, export, 27-voxel NN -- CUDA path (through the C ABI)
vs the FP64 CPU oracle, element by element, bit-exact (integer / byte / index work)."""
import numpy as np
import pytest
import torch

import far_scenes as scenes
import oracle
from helpers import load_golden, np_pack, np_voxel_index

pytestmark = pytest.mark.gpu

far = pytest.importorskip("paper_2606_26010_b200")


def _cloud(rng, n, scale=20.0, clustered=True):
    pts = rng.uniform(-scale, scale, size=(n, 3))
    if clustered:   # a dense blob so that caps are hit
        m = n // 3
        pts[:m] = rng.normal(0.0, 0.6, size=(m, 3)) + np.array([3.0, -2.0, 1.0])
    return pts.astype(np.float32)


def _assert_same_map(g, o, with_cov=False):
    assert np.array_equal(g["keys"], o["keys"])
    assert np.array_equal(g["counts"], o["counts"])
    assert np.array_equal(g["ids"], o["ids"])
    assert np.array_equal(g["xyz"].view(np.uint32), o["xyz"].view(np.uint32))   # bit-exact coordinates
    if with_cov:
        assert np.array_equal(g["cov_valid"], o["cov_valid"])
        v = o["cov_valid"].astype(bool)
        a, b = g["cov"][v].astype(np.float64), o["cov"][v].astype(np.float64)
        rel = np.linalg.norm(a - b, axis=1) / np.linalg.norm(b, axis=1)
        assert rel.max() < 1e-4 if len(rel) else True


# ---- A1 ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("voxel", [0.25, 0.5, 1.0, 2.0, 4.0, 0.3])
def test_voxel_keys_bit_exact(voxel):
    rng = np.random.default_rng(11)
    pts = _cloud(rng, 100_003, scale=300.0)
    pts[5] = [np.nan, 0, 0]
    pts[6] = [0, np.inf, 0]
    pts[7] = [3e7, 0, 0]            # voxel index out of +-2^20
    pts[8] = [-0.0, 0.5, -0.5]
    k_o, v_o = oracle.keys(pts, voxel)
    k_g = far.voxel_keys(pts, voxel).cpu().numpy().view(np.uint64)
    assert np.array_equal(k_g, k_o)
    assert np.array_equal(k_g != np.uint64(0xFFFFFFFFFFFFFFFF), v_o)


def test_voxel_keys_golden_and_stride4():
    g = load_golden("key_examples.json")
    for k3, hx in g["pack_cases"]:
        k = np.array(k3, dtype=np.float64)
        p = ((k + 0.5) * g["voxel"]).astype(np.float32)[None, :]       # voxel centre: exactly representable
        p4 = np.concatenate([p, np.ones((1, 1), np.float32)], axis=1)
        for arr in (p, p4):
            got = int(far.voxel_keys(arr, g["voxel"]).cpu().numpy().view(np.uint64)[0])
            assert got == int(hx, 16)
    for x, want in g["floor_cases"]:
        key = int(far.voxel_keys(np.array([[x, 0.0, 0.0]], dtype=np.float32), g["voxel"]).cpu().numpy().view(np.uint64)[0])
        assert oracle.unpack_key(key)[0] == want


# ---- A2 ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n,voxel", [(0, 1.0), (1, 1.0), (1023, 0.5), (1024, 0.5), (1025, 1.0), (77_777, 1.0), (300_000, 0.5)])
def test_voxelize_bit_exact(n, voxel):
    rng = np.random.default_rng(n + 1)
    pts = _cloud(rng, n, scale=40.0)
    if n > 10:
        pts[3] = np.nan
        pts[n // 2] = np.inf
    o_xyz, o_idx = oracle.voxelize(pts, voxel) if n else (np.zeros((0, 3), np.float32), np.zeros(0, np.int32))
    g_xyz, g_idx = far.voxelize(pts, voxel) if n else far.Voxelizer(8)(torch.zeros((0, 3), device="cuda"), voxel)
    assert np.array_equal(g_idx.cpu().numpy(), o_idx)
    assert np.array_equal(g_xyz.cpu().numpy().view(np.uint32), o_xyz.view(np.uint32))


def test_voxelize_lidar_scan_and_idempotence():
    c2 = scenes.c2_single_frame(seed=1, n_map_candidates=1000, rings=16, azimuths=512)
    scan = c2["scan"]
    o_xyz, o_idx = oracle.voxelize(scan, 1.0)
    g_xyz, g_idx = far.voxelize(scan, 1.0)
    assert np.array_equal(g_idx.cpu().numpy(), o_idx)
    again, idx2 = far.voxelize(g_xyz, 1.0)
    assert torch.equal(again, g_xyz) and np.array_equal(idx2.cpu().numpy(), np.arange(len(o_idx)))


# ---- A3/A4 ------------------------------------------------------------------------------------------------
def test_insert_golden_example():
    g = load_golden("insert_worked_example.json")
    m = far.Map(g["voxel"], g["cap"], 64)
    st = m.insert(np.array(g["points"], dtype=np.float32))
    e = m.export()
    got = {int(k): [int(i) for i in e["ids"][v, :e["counts"][v]]] for v, k in enumerate(e["keys"])}
    want = {oracle.pack_key(*map(int, k.split(","))): ids for k, ids in g["expect"].items()}
    assert got == want
    assert st["n_accepted"] == 3 and st["n_new_voxels"] == 2 and st["n_offered"] == 4


@pytest.mark.parametrize("cap", [1, 4, 20, 33, 40])
def test_insert_contents_bit_exact(cap):
    rng = np.random.default_rng(100 + cap)
    pts = _cloud(rng, 60_001, scale=15.0)
    pts[17] = np.nan
    mo = oracle.Map(0.5, cap)
    mg = far.Map(0.5, cap, 200_000)
    so = mo.insert(pts)
    sg = mg.insert(pts)
    assert sg == so
    _assert_same_map(mg.export(), mo.export())
    assert mg.size() == mo.size()


def test_insert_batch_invariance_and_internal_chunking():
    rng = np.random.default_rng(7)
    pts = _cloud(rng, 50_000, scale=10.0)
    mo = oracle.Map(0.5, 20)
    so = mo.insert(pts)
    ref = mo.export()
    # many external batches of ragged sizes
    mg = far.Map(0.5, 20, 100_000)
    cuts = [0, 1, 33, 1000, 1001, 20_000, 49_999, 50_000]
    for a, b in zip(cuts[:-1], cuts[1:]):
        mg.insert(pts[a:b])
    _assert_same_map(mg.export(), ref)
    # one call that the library has to chunk internally (max_batch smaller than n)
    mc = far.Map(0.5, 20, 100_000, max_batch=4096)
    st = mc.insert(pts)
    assert st == so
    _assert_same_map(mc.export(), ref)


def test_insert_with_pose_bit_exact_and_device_pose():
    rng = np.random.default_rng(8)
    pts = _cloud(rng, 30_000, scale=50.0)
    T = scenes.pose_from_rpy_t(0.03, -0.02, 0.7, [12.5, -3.25, 0.8])
    mo = oracle.Map(1.0, 20)
    so = mo.insert(pts, pose=T)
    mg = far.Map(1.0, 20, 100_000)
    sg = mg.insert(pts, pose=T)
    assert sg == so
    _assert_same_map(mg.export(), mo.export())
    # same through the device-pose entry point
    md = far.Map(1.0, 20, 100_000)
    d_pose = torch.frombuffer(bytearray(bytes(far.Pose.from_rt(T))), dtype=torch.uint8).cuda()
    md.insert_enqueue(pts, d_pose=d_pose)
    _assert_same_map(md.export(), mo.export())


def test_insert_stride4_and_invalid_points_consume_ids():
    rng = np.random.default_rng(9)
    pts = _cloud(rng, 5000, scale=5.0)
    pts[10] = np.nan
    pts[11, 2] = -np.inf
    p4 = np.concatenate([pts, rng.normal(size=(5000, 1)).astype(np.float32)], axis=1)
    mo = oracle.Map(0.5, 20)
    so = mo.insert(p4)
    mg = far.Map(0.5, 20, 20_000)
    sg = mg.insert(p4)
    assert sg == so and sg["n_invalid"] == 2
    _assert_same_map(mg.export(), mo.export())
    assert mg.size()[2] == 5000


def test_insert_is_deterministic_across_runs():
    rng = np.random.default_rng(10)
    pts = torch.as_tensor(_cloud(rng, 200_000, scale=6.0)).cuda()
    exports = []
    for _ in range(3):
        m = far.Map(0.5, 20, 50_000)
        m.insert(pts)
        exports.append(m.export())
        m.close()
    for e in exports[1:]:
        _assert_same_map(e, exports[0])


def test_table_full_is_reported_not_fatal():
    """FAR_ERR_FULL (far.h): the bucket pool is an exact limit; excess NEW voxels are dropped and counted; the status is
    raised on the device, mirrored into pinned host memory and returned by later calls without a sync; pruning clears it."""
    rng = np.random.default_rng(12)
    pts = _cloud(rng, 20_000, scale=50.0, clustered=False)
    m = far.Map(0.5, 4, 1000)       # far fewer voxels than the cloud occupies
    assert m.status() == far.OK
    st = m.insert(pts)              # reads the statistics back: the kernels have run
    assert st["n_dropped_full"] > 0 and st["n_new_voxels"] == 1000
    assert st["n_accepted"] + st["n_dropped_full"] + st["n_invalid"] <= st["n_offered"]
    s = m.stats()
    assert s["n_voxels"] == 1000 and s["full"] == 1 and s["n_fresh_buckets"] == 0
    assert m.status() == far.ERR_FULL
    rc = far.lib().far_map_insert(m._h, None, 0, 3, None, 0, None, None)     # the C call itself reports it
    assert rc == far.ERR_FULL
    e = m.export()
    assert (e["counts"] <= 4).all() and (e["counts"] >= 1).all() and len(e["keys"]) == 1000
    # every stored voxel holds exactly what the oracle stores for it (which voxels were dropped is unspecified, R3)
    mo = oracle.Map(0.5, 4)
    mo.insert(pts)
    eo = mo.export()
    pos = np.searchsorted(eo["keys"], e["keys"])
    assert np.array_equal(eo["keys"][pos], e["keys"]) and np.array_equal(eo["ids"][pos], e["ids"])
    # pruning frees buckets: the flag clears and new voxels are accepted again
    pr = m.prune([0.0, 0.0, 0.0], 20.0)
    assert pr["n_voxels_removed"] > 0
    assert m.status() == far.OK and m.stats()["full"] == 0
    near = (rng.uniform(-5, 5, size=(pr["n_voxels_removed"] // 4, 3)) + np.array([30.0, 30.0, 30.0])).astype(np.float32)
    st2 = m.insert(near)
    assert st2["n_dropped_full"] == 0 and st2["n_new_voxels"] > 0 and not m.full_seen


# ---- A5 ---------------------------------------------------------------------------------------------------
def test_prune_matches_oracle_and_reinsert():
    rng = np.random.default_rng(13)
    pts = _cloud(rng, 80_000, scale=30.0)
    mo, mg = oracle.Map(1.0, 20), far.Map(1.0, 20, 200_000)
    mo.insert(pts); mg.insert(pts)
    c = [1.5, -2.0, 0.25]
    assert mg.prune(c, 1e9) == mo.prune(c, 1e9)          # no-op
    so, sg = mo.prune(c, 17.3), mg.prune(c, 17.3)
    assert sg == so and sg["n_voxels_removed"] > 0
    _assert_same_map(mg.export(), mo.export())
    # pruned voxels come back empty: re-insert a second cloud over the whole region
    more = _cloud(rng, 40_000, scale=30.0)
    assert mg.insert(more) == mo.insert(more)
    _assert_same_map(mg.export(), mo.export())
    st = mg.stats()
    assert st["n_voxels"] == mo.size()[0] and st["n_points"] == mo.size()[1]
    # prune by a device-resident pose gives the same result
    T = (np.eye(3), np.array(c))
    d_pose = torch.frombuffer(bytearray(bytes(far.Pose.from_rt(T))), dtype=torch.uint8).cuda()
    mg.prune_enqueue(radius=9.0, d_pose=d_pose)
    mo.prune(c, 9.0)
    _assert_same_map(mg.export(), mo.export())


def test_dead_keys_rehash_and_clear_keep_contents_semantics():
    rng = np.random.default_rng(14)
    pts = _cloud(rng, 60_000, scale=30.0)
    mo, mg = oracle.Map(1.0, 20), far.Map(1.0, 20, 200_000, with_cov=True)
    mo.insert(pts, compute_cov=True); mg.insert(pts, compute_cov=True)
    n_live0 = mg.stats()["n_voxels"]
    # a small prune leaves dead keys behind (below the rebuild threshold 32 + live / 8): absent for every query, re-usable
    assert mo.prune([0, 0, 0], 49.0) == mg.prune([0, 0, 0], 49.0)
    st = mg.stats()
    assert 0 < st["n_dead_keys"] < 32 + st["n_voxels"] // 8 and st["n_rehash"] == 0
    assert st["n_free_buckets"] == st["n_dead_keys"] and st["n_keys"] == n_live0
    _assert_same_map(mg.export(with_cov=True), mo.export(with_cov=True), with_cov=True)
    q = _cloud(rng, 5000, scale=32.0)
    ids_o, d2_o = mo.nn(q)
    ids_g, d2_g = mg.nn(q)
    assert np.array_equal(ids_g.cpu().numpy().view(np.uint32), ids_o)
    # a large prune passes the threshold: the prune call rebuilds the table itself (no dead keys afterwards)
    assert mo.prune([0, 0, 0], 20.0) == mg.prune([0, 0, 0], 20.0)
    st = mg.stats()
    assert st["n_dead_keys"] == 0 and st["n_rehash"] == 1 and st["n_voxels"] == mo.size()[0] and st["n_keys"] == st["n_voxels"]
    _assert_same_map(mg.export(with_cov=True), mo.export(with_cov=True), with_cov=True)
    ids_o, d2_o = mo.nn(q)
    ids_g, d2_g = mg.nn(q)
    assert np.array_equal(ids_g.cpu().numpy().view(np.uint32), ids_o)
    assert np.array_equal(d2_g.cpu().numpy().view(np.uint32), d2_o.view(np.uint32))
    # freed buckets are re-used by later inserts (new voxels and re-created ones), contents still the oracle's
    more = _cloud(rng, 30_000, scale=30.0)
    assert mg.insert(more, compute_cov=True) == mo.insert(more, compute_cov=True)
    _assert_same_map(mg.export(with_cov=True), mo.export(with_cov=True), with_cov=True)
    # explicit rehash with a few dead keys
    assert mo.prune([1, 0, 0], 29.0) == mg.prune([1, 0, 0], 29.0)
    mg.rehash()
    st = mg.stats()
    assert st["n_dead_keys"] == 0 and st["n_keys"] == st["n_voxels"] == mo.size()[0]
    _assert_same_map(mg.export(), mo.export())
    mg.clear()
    assert mg.size() == (0, 0, 0)
    mo2 = oracle.Map(1.0, 20)
    mo2.insert(pts[:1000]); mg.insert(pts[:1000])
    _assert_same_map(mg.export(), mo2.export())


def test_renumber_matches_oracle_and_keeps_order():
    """R22: ids -= smallest live id (also triggered automatically every `renumber_every` offered points)"""
    rng = np.random.default_rng(15)
    mo, mg = oracle.Map(1.0, 8), far.Map(1.0, 8, 100_000, renumber_every=50_000)
    offered_since = 0
    for b in range(12):
        pts = (rng.uniform(-10, 10, size=(20_000, 3)) + np.array([8.0 * b, 0, 0])).astype(np.float32)
        if offered_since > 0 and offered_since + len(pts) > 50_000:       # the library's deterministic trigger, restated
            mo.renumber()
            offered_since = 0
        assert mg.insert(pts) == mo.insert(pts)
        offered_since += len(pts)
        c = [8.0 * b, 0.0, 0.0]
        assert mg.prune(c, 12.0) == mo.prune(c, 12.0)
        assert mg.size() == mo.size(), b
    assert mo.size()[2] < 12 * 20_000                                  # the counter really was pulled back
    _assert_same_map(mg.export(), mo.export())
    sub = mo.renumber()
    mg.renumber()
    assert sub > 0 and mg.size() == mo.size()
    e = mg.export()
    _assert_same_map(e, mo.export())
    assert e["ids"][e["counts"][:, None] > np.arange(8)[None, :]].min() == 0
    q = (rng.uniform(-10, 10, size=(3000, 3)) + np.array([88.0, 0, 0])).astype(np.float32)
    ids_g, _ = mg.nn(q)
    assert np.array_equal(ids_g.cpu().numpy().view(np.uint32), mo.nn(q)[0])
    mg.prune([0, 0, 0], 1.0); mo.prune([0, 0, 0], 1.0)                  # empties the map
    mg.renumber(); mo.renumber()
    assert mg.size() == mo.size() == (0, 0, 0)


def test_sliding_window_5000_frames_never_fills_and_matches_oracle():
    """PAPER.md:109 prunes every frame, :171,186 nothing may allocate: a 200 m window slides for 5,000 frames through a map
    sized for the window only.  Buckets are recycled through the free list, dead keys are dropped by the prune calls'
    own rebuilds, ids are renumbered on the way; the map never reports full and ends equal to the oracle's."""
    rng = np.random.default_rng(16)
    v, cap, step, radius, n_pts, frames = 1.0, 20, 7.0, 100.0, 1500, 5000
    mo = oracle.Map(v, cap)
    mg = far.Map(v, cap, 40_000, max_batch=4096, renumber_every=1_000_000)
    assert mg.stats()["n_slots"] == 131072
    offered_since, peak_dead, peak_live = 0, 0, 0
    q0 = None
    t_nn = {}

    def time_nn(center):
        q = torch.as_tensor((rng.uniform(-1, 1, size=(200_000, 3)) * np.array([90.0, 12.0, 3.0]) + center).astype(np.float32)).cuda()
        ts = []
        for _ in range(7):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); mg.nn(q); b.record(); torch.cuda.synchronize()
            ts.append(a.elapsed_time(b))
        return float(np.median(ts[2:]))

    for f in range(frames):
        c = np.array([step * f, 0.0, 0.0])
        # a corridor-shaped "scan": points up to 95 m ahead of and behind the sensor, 24 m wide, 6 m high
        pts = (rng.uniform(-1, 1, size=(n_pts, 3)) * np.array([95.0, 12.0, 3.0]) + c).astype(np.float32)
        if offered_since > 0 and offered_since + n_pts > 1_000_000:
            mo.renumber()
            offered_since = 0
        mo.insert(pts)
        mg.insert_enqueue(pts)
        offered_since += n_pts
        mo.prune(c, radius)
        mg.prune_enqueue(c, radius)
        if f % 250 == 249 or f == frames - 1:
            st = mg.stats()
            assert st["full"] == 0 and mg.status() == far.OK, f
            assert (st["n_voxels"], st["n_points"], st["next_id"]) == mo.size(), f
            peak_dead, peak_live = max(peak_dead, st["n_dead_keys"]), max(peak_live, st["n_voxels"])
            assert st["n_dead_keys"] < 64 + st["n_voxels"] // 4, (f, st)
            assert st["n_keys"] == st["n_voxels"] + st["n_dead_keys"]
        if f in (249, frames - 1):
            t_nn[f] = time_nn(c)
    st = mg.stats()
    assert st["n_rehash"] > 50 and peak_live <= 40_000 and mo.size()[2] < 2_500_000
    _assert_same_map(mg.export(), mo.export())
    # lookups are as fast at the end as at the start: dead keys and probe bounds do not accumulate
    assert t_nn[frames - 1] < 1.15 * t_nn[249], t_nn


# ---- A6 ---------------------------------------------------------------------------------------------------
def test_nn_golden_example():
    g = load_golden("nn_worked_example.json")
    m = far.Map(g["voxel"], 20, 64)
    m.insert(np.array(g["stored"], dtype=np.float32))
    for case in g["queries"]:
        ids, d2 = m.nn(np.array([case["q"]], dtype=np.float32))
        assert int(ids.cpu().numpy().view(np.uint32)[0]) == case["id"]
        want = np.inf if case["d2"] == "inf" else case["d2"]
        assert float(d2[0]) == pytest.approx(want, rel=1e-6)
    t = g["tie"]
    m2 = far.Map(g["voxel"], 20, 64)
    m2.insert(np.array(t["stored"], dtype=np.float32))
    ids, _ = m2.nn(np.array([t["q"]], dtype=np.float32))
    assert int(ids[0]) == t["id"]


@pytest.mark.parametrize("voxel,cap", [(0.25, 20), (0.5, 20), (1.0, 20), (2.0, 20), (4.0, 40), (1.0, 1)])
def test_nn_bit_exact(voxel, cap):
    rng = np.random.default_rng(int(voxel * 100) + cap)
    pts = _cloud(rng, 120_000, scale=25.0)
    mo, mg = oracle.Map(voxel, cap), far.Map(voxel, cap, 400_000)
    mo.insert(pts); mg.insert(pts)
    q = np.concatenate([pts[rng.integers(0, len(pts), 20_000)] + rng.normal(0, 0.1, (20_000, 3)).astype(np.float32),
                        rng.uniform(-40, 40, (10_001, 3)).astype(np.float32)]).astype(np.float32)
    q[5] = np.nan
    ids_o, d2_o = mo.nn(q, nthreads=8)
    ids_g, d2_g = mg.nn(q)
    assert np.array_equal(ids_g.cpu().numpy().view(np.uint32), ids_o)
    assert np.array_equal(d2_g.cpu().numpy().view(np.uint32), d2_o.view(np.uint32))
    assert (ids_o == oracle.NO_ID).any() and (ids_o != oracle.NO_ID).any()


def test_nn_exact_ties_break_to_lowest_id():
    # lattice points: many exactly equidistant candidates
    g = np.stack(np.meshgrid(np.arange(-8, 8), np.arange(-8, 8), np.arange(-2, 2), indexing="ij"), -1).reshape(-1, 3)
    pts = (g * 0.25).astype(np.float32)
    rng = np.random.default_rng(3)
    pts = pts[rng.permutation(len(pts))]
    mo, mg = oracle.Map(0.5, 20), far.Map(0.5, 20, 10_000)
    mo.insert(pts); mg.insert(pts)
    q = (g[::3] * 0.25 + 0.125).astype(np.float32)          # cell centres: 8 equidistant corners
    ids_o, d2_o = mo.nn(q)
    ids_g, d2_g = mg.nn(q)
    assert np.array_equal(ids_g.cpu().numpy().view(np.uint32), ids_o)
    assert np.array_equal(d2_g.cpu().numpy(), d2_o)


def test_empty_calls():
    m = far.Map(0.5, 20, 1024, with_cov=True)
    z = torch.zeros((0, 3), device="cuda")
    assert m.insert(z)["n_offered"] == 0
    ids, d2 = m.nn(z)
    assert ids.numel() == 0
    ids, d2 = m.nn(np.array([[0.1, 0.2, 0.3]], dtype=np.float32))      # empty map
    assert int(ids.cpu().numpy().view(np.uint32)[0]) == far.NO_ID and np.isinf(float(d2[0]))
    cov, valid = m.knn_cov(np.array([[0.1, 0.2, 0.3]], dtype=np.float32))
    assert int(valid[0]) == 0 and cov[0].tolist() == [1, 0, 0, 1, 0, 1]
    assert m.export()["keys"].size == 0
    assert m.prune([0, 0, 0], 1.0) == dict(n_voxels_removed=0, n_points_removed=0, n_voxels_left=0, n_points_left=0)


def test_dead_key_count_follows_revived_and_bucketless_keys():
    """The table is rebuilt (in-place rehash inside far_map_prune) when the keys that own no bucket stop being a small
    fraction of the live ones.  That count has to follow the table: a pruned voxel that is opened again is no longer dead,
    and a key claimed while the bucket pool was exhausted is dead from the start.
    (a) a vehicle going back and forth over the same ground: each lap prunes and re-opens the same ~8 % of the voxels; no
        lap leaves more dead keys than the first one did, so no lap may trigger a rebuild;
    (b) a map whose pool ran out: the bucket-less keys are reclaimed by the next prune even if it removes nothing."""
    rng = np.random.default_rng(41)
    # (a) 12,000 voxels on a 0.5 m lattice plane, one point each; the strip x < 4 m holds 960 of them (8 %)
    ij = np.stack(np.meshgrid(np.arange(100), np.arange(120), indexing="ij"), axis=-1).reshape(-1, 2)
    pts = np.concatenate([ij * 0.5 + 0.25, np.full((len(ij), 1), 0.25)], axis=1).astype(np.float32)
    pts = pts[rng.permutation(len(pts))]
    mo, mg = oracle.Map(0.5, 4), far.Map(0.5, 4, 20_000)
    assert mg.insert(pts) == mo.insert(pts)
    centre, radius = [1000.0, 30.0, 0.25], 996.0          # keeps x >= 4 m, up to the curvature of a 1 km circle
    strip = None
    for lap in range(6):
        assert mg.prune(centre, radius) == mo.prune(centre, radius)
        if strip is None:                                # the points of the voxels the prune removes: the same every lap
            gone = ~np.isin(np_pack(np_voxel_index(pts, 0.5)), mo.export()["keys"])
            strip = pts[gone]
            assert 900 < len(strip) < 1100
        s = mg.stats()
        assert 800 < s["n_dead_keys"] < 32 + s["n_voxels"] // 8, s
        assert s["n_rehash"] == 0, (lap, s)
        assert mg.insert(strip) == mo.insert(strip)
        s = mg.stats()
        assert s["n_dead_keys"] == 0 and s["n_voxels"] == 12_000 and s["n_keys"] == 12_000, s
        _assert_same_map(mg.export(), mo.export())
    # one more prune, now of a larger part (x < 12 m, 24 %): the rebuild is due and happens
    assert mg.prune(centre, 988.0) == mo.prune(centre, 988.0)
    s = mg.stats()
    assert s["n_rehash"] == 1 and s["n_dead_keys"] == 0 and s["n_keys"] == s["n_voxels"], s
    _assert_same_map(mg.export(), mo.export())
    # (b) 1,000 buckets, a cloud that wants ~15,000 voxels
    m = far.Map(0.5, 4, 1000)
    st = m.insert(_cloud(rng, 20_000, scale=50.0, clustered=False))
    assert st["n_new_voxels"] == 1000 and st["n_dropped_full"] > 0
    s = m.stats()
    assert s["n_dead_keys"] > 0 and s["n_keys"] == 1000 + s["n_dead_keys"], s
    before = m.export()
    assert m.prune([0.0, 0.0, 0.0], 1e4)["n_voxels_removed"] == 0
    s = m.stats()
    assert s["n_rehash"] == 1 and s["n_dead_keys"] == 0 and s["n_keys"] == 1000 and s["n_voxels"] == 1000, s
    _assert_same_map(m.export(), before)


def test_snapshot_restore_brings_back_the_full_status():
    """far_map_status / the return code of insert are served from a host-visible mirror of the device's sticky full flag
    (far.h).  Restoring a snapshot taken BEFORE the map filled up must bring that mirror back with the counters: the
    restored map has free buckets and says so; and it can fill up (and say so) again."""
    rng = np.random.default_rng(31)
    few = (rng.uniform(-3, 3, size=(200, 3))).astype(np.float32)
    many = _cloud(rng, 20_000, scale=50.0, clustered=False)
    m = far.Map(0.5, 4, 1000)
    m.insert(few)
    assert m.status() == far.OK
    snap = m.snapshot()
    before = m.export()
    assert m.insert(many)["n_dropped_full"] > 0
    assert m.status() == far.ERR_FULL and m.stats()["full"] == 1
    m.restore(snap)
    torch.cuda.synchronize()
    assert m.stats()["full"] == 0 and m.status() == far.OK
    assert far.lib().far_map_insert(m._h, None, 0, 3, None, 0, None, None) == far.OK
    _assert_same_map(m.export(), before)
    assert m.insert(many)["n_dropped_full"] > 0 and m.status() == far.ERR_FULL
    # ... and the other way round: a snapshot of a FULL map restored onto the map after pruning made room
    full_snap = m.snapshot()
    assert m.prune([0.0, 0.0, 0.0], 10.0)["n_voxels_removed"] > 0 and m.status() == far.OK
    m.restore(full_snap)
    torch.cuda.synchronize()
    assert m.status() == far.ERR_FULL and m.stats()["full"] == 1
    far.Map.snapshot_destroy(snap); far.Map.snapshot_destroy(full_snap)


def test_id_range_check_survives_a_renumber_undone_by_a_restore():
    """R3/R22 at the top of the u32 id range (FAR_ERR_RANGE, far.h).  Ids advance by the points OFFERED, so 3 x 2^30 rows
    of NaN take the counter to 3.2e9 without storing anything.  A renumber pass enqueued after a snapshot reports a small
    counter to the host; restoring the snapshot puts the large counter back, and the host-side bound must not fold that
    stale report: the next 2^30-row insert would wrap the ids past 2^32 and has to be refused, nothing inserted.  After an
    explicit renumber of the restored map the same insert goes through and the ids are the renumbered ones."""
    big = 1 << 30
    nan = torch.full((big, 3), float("nan"), dtype=torch.float32, device="cuda")      # 12.9 GB of invalid rows
    L, st = far.lib(), far._stream()

    def offer_nan():
        return L.far_map_insert(m._h, far._ptr(nan), big, 3, None, 0, None, st)

    rng = np.random.default_rng(32)
    m = far.Map(1.0, 8, 10_000)
    anchor = np.array([[500.5, 500.5, 0.5]], dtype=np.float32)        # id 0 stays alive: automatic renumbering subtracts 0
    assert m.insert(anchor)["n_accepted"] == 1
    for _ in range(3):
        assert offer_nan() == far.OK
    pts = (rng.uniform(-4, 4, size=(1000, 3))).astype(np.float32)
    first = 1 + 3 * big
    assert m.insert(pts)["n_accepted"] > 900
    assert m.size()[2] == first + 1000
    e = m.export()
    live = np.sort(e["ids"][e["ids"] != far.NO_ID].astype(np.int64))
    assert live[0] == 0 and live[1] == first and live[-1] <= first + 999
    assert m.prune([0.0, 0.0, 0.0], 50.0)["n_voxels_removed"] == 1    # the anchor goes: smallest live id is now ~3.2e9
    snap = m.snapshot()
    m.renumber()
    torch.cuda.synchronize()                                         # the pass has reported next_id = 1000 to the host
    assert m.size()[2] == 1000
    m.restore(snap)
    assert m.size()[2] == first + 1000
    assert offer_nan() == far.ERR_RANGE                              # 3.2e9 + 1001 + 2^30 > 2^32 - 1
    assert m.size()[2] == first + 1000                               # nothing was offered
    m.renumber()
    assert offer_nan() == far.OK
    assert m.size()[2] == 1000 + big
    e2 = m.export()
    live2 = np.sort(e2["ids"][e2["ids"] != far.NO_ID].astype(np.int64))
    assert np.array_equal(live2, live[1:] - first)
    far.Map.snapshot_destroy(snap)


def test_snapshot_restore_count27_and_launch_accounting():
    rng = np.random.default_rng(21)
    pts = _cloud(rng, 40_000, scale=12.0)
    mo, mg = oracle.Map(0.5, 20), far.Map(0.5, 20, 100_000, with_cov=True)
    mo.insert(pts[:20_000], compute_cov=True); mg.insert(pts[:20_000], compute_cov=True)
    snap = mg.snapshot()
    before = mg.export(with_cov=True)
    n0 = far.launch_count()
    mg.insert(pts[20_000:], compute_cov=True)
    mg.prune([0, 0, 0], 5.0)
    assert far.launch_count() - n0 >= 5            # claim, commit, knn_cov, stats, prune, ...
    mg.restore(snap)
    after = mg.export(with_cov=True)
    for k in ("keys", "counts", "ids", "xyz", "cov", "cov_valid"):
        assert np.array_equal(before[k].view(np.uint8), after[k].view(np.uint8)), k
    assert mg.size() == mo.size()
    # the restored map continues exactly like the oracle (ids continue from the snapshot's counter)
    assert mg.insert(pts[20_000:]) == mo.insert(pts[20_000:])
    _assert_same_map(mg.export(), mo.export())
    far.Map.snapshot_destroy(snap)
    # count27 = number of candidates the 27-voxel search scans, checked against the oracle's k-NN list length
    q = pts[:500]
    cnt = mg.count27(q).cpu().numpy()
    ids, _ = mo.knn(q, 27 * 20)
    assert np.array_equal(cnt, (ids != oracle.NO_ID).sum(axis=1))
    # per-kernel timing facility
    far.profile_enable(True)
    mg.nn(q)
    far.profile_enable(False)
    prof = far.profile_collect()
    assert "nn_kernel" in prof and prof["nn_kernel"][1] == 1 and prof["nn_kernel"][0] > 0
