"""Property tests (hypothesis) on small adversarial clouds: coordinates on a coarse lattice so that points coincide, sit
exactly on voxel faces and tie in distance; tiny caps so that the cap binds; arbitrary batch splits.

CPU part (`-m "not gpu"`): invariants of the oracle that hold by the definitions in DESIGN.md (R2, R3, R5, R6) and are
checked against NumPy restatements.  GPU part (`-m gpu`): the same drawn inputs through the CUDA path must equal the
oracle bit for bit (tier 3).
"""
import numpy as np
import pytest
from hypothesis import HealthCheck, given, settings, strategies as st

import oracle
from helpers import np_capped_contents, np_nn_bruteforce, np_pack, np_voxel_index

SET = dict(deadline=None, suppress_health_check=[HealthCheck.too_slow, HealthCheck.data_too_large])


@st.composite
def clouds(draw, max_n=400):
    n = draw(st.integers(0, max_n))
    step = draw(st.sampled_from([0.25, 0.5, 1.0]))                  # lattice pitch: many exact coincidences and face hits
    span = draw(st.integers(2, 12))
    seed = draw(st.integers(0, 2**31 - 1))
    rng = np.random.default_rng(seed)
    pts = (rng.integers(-span, span + 1, size=(n, 3)) * step).astype(np.float32)
    jitter = draw(st.booleans())
    if jitter and n:
        pts += rng.normal(0, 0.05, pts.shape).astype(np.float32)
    return pts


voxels = st.sampled_from([0.25, 0.5, 1.0, 2.0])
caps = st.integers(1, 6)


def _contents(exp):
    return {int(k): [int(i) for i in exp["ids"][v, :exp["counts"][v]]] for v, k in enumerate(exp["keys"])}


# ------------------------------------------------------------------------------------------------- oracle (CPU)
@settings(max_examples=60, **SET)
@given(clouds(), voxels, caps, st.lists(st.integers(0, 400), max_size=4))
def test_oracle_insert_is_batch_invariant_and_capped(pts, voxel, cap, cuts):
    one = oracle.Map(voxel, cap)
    one.insert(pts)
    many = oracle.Map(voxel, cap)
    edges = sorted({0, len(pts), *[min(c, len(pts)) for c in cuts]})
    for a, b in zip(edges, edges[1:]):
        many.insert(pts[a:b])
    e1, e2 = one.export(), many.export()
    assert np.array_equal(e1["keys"], e2["keys"]) and np.array_equal(e1["ids"], e2["ids"])
    assert np.array_equal(e1["xyz"].view(np.uint32), e2["xyz"].view(np.uint32))
    assert (e1["counts"] <= cap).all()
    want = np_capped_contents(pts, voxel, cap) if len(pts) else {}   # first `cap` indices per key, ascending
    assert _contents(e1) == want


@settings(max_examples=40, **SET)
@given(clouds(), voxels)
def test_oracle_voxelize_is_first_point_per_voxel_and_idempotent(pts, voxel):
    ds, idx = oracle.voxelize(pts, voxel)
    keys = np_pack(np_voxel_index(pts, voxel)) if len(pts) else np.zeros(0, np.uint64)
    _, first = np.unique(keys, return_index=True)
    assert np.array_equal(idx, np.sort(first))
    ds2, idx2 = oracle.voxelize(ds, voxel)
    assert np.array_equal(ds2.view(np.uint32), ds.view(np.uint32)) and np.array_equal(idx2, np.arange(len(ds)))


@settings(max_examples=40, **SET)
@given(clouds(max_n=250), voxels, caps, clouds(max_n=40))
def test_oracle_nn_is_the_lexicographic_minimum_over_the_27_voxels(pts, voxel, cap, q):
    m = oracle.Map(voxel, cap)
    m.insert(pts)
    if len(q) == 0:
        return
    ids, d2 = m.nn(q)
    e = m.export()
    stored = e["counts"][:, None] > np.arange(cap)[None, :]
    bf_ids, bf_d2 = np_nn_bruteforce(e["xyz"][stored], e["ids"][stored], q, voxel)
    assert np.array_equal(ids, bf_ids)
    assert np.array_equal(d2, bf_d2.astype(np.float32))


@settings(max_examples=40, **SET)
@given(clouds(), voxels, caps, st.floats(0.0, 8.0), st.tuples(st.floats(-3, 3), st.floats(-3, 3), st.floats(-3, 3)))
def test_oracle_prune_removes_exactly_the_far_voxels(pts, voxel, cap, radius, centre):
    m = oracle.Map(voxel, cap)
    m.insert(pts)
    before = m.export()
    st_ = m.prune(centre, radius)
    after = m.export()
    from helpers import np_unpack
    k = np_unpack(before["keys"]) if len(before["keys"]) else np.zeros((0, 3))
    d2 = (((k + 0.5) * voxel - np.asarray(centre)) ** 2).sum(axis=1) if len(k) else np.zeros(0)
    keep = d2 <= radius * radius
    assert np.array_equal(after["keys"], before["keys"][keep])
    assert st_["n_voxels_removed"] == int((~keep).sum()) and st_["n_points_removed"] == int(before["counts"][~keep].sum())


# ------------------------------------------------------------------------------------------------- CUDA path (GPU)
gpu = pytest.mark.gpu


def _far():
    import paper_2606_26010_b200 as far
    return far


@gpu
@settings(max_examples=40, **SET)
@given(clouds(max_n=3000), voxels, caps, st.lists(st.integers(0, 3000), max_size=3))
def test_gpu_insert_export_equal_oracle_under_any_batching(pts, voxel, cap, cuts):
    far = _far()
    mo, mg = oracle.Map(voxel, cap), far.Map(voxel, cap, 1 << 13)
    edges = sorted({0, len(pts), *[min(c, len(pts)) for c in cuts]})
    for a, b in zip(edges, edges[1:]):
        assert mg.insert(pts[a:b]) == mo.insert(pts[a:b])
    eg, eo = mg.export(), mo.export()
    assert np.array_equal(eg["keys"], eo["keys"]) and np.array_equal(eg["counts"], eo["counts"])
    assert np.array_equal(eg["ids"], eo["ids"]) and np.array_equal(eg["xyz"].view(np.uint32), eo["xyz"].view(np.uint32))
    mg.close()


@gpu
@settings(max_examples=40, **SET)
@given(clouds(max_n=2000), voxels, caps, clouds(max_n=300))
def test_gpu_nn_and_voxelize_equal_oracle_with_ties_and_coincident_points(pts, voxel, cap, q):
    far = _far()
    mo, mg = oracle.Map(voxel, cap), far.Map(voxel, cap, 1 << 13)
    mo.insert(pts); mg.insert(pts)
    if len(q):
        ids_o, d2_o = mo.nn(q)
        ids_g, d2_g = mg.nn(q)
        assert np.array_equal(ids_g.cpu().numpy().view(np.uint32), ids_o)
        assert np.array_equal(d2_g.cpu().numpy().view(np.uint32), d2_o.view(np.uint32))
    if len(pts):
        ds_o, idx_o = oracle.voxelize(pts, voxel)
        ds_g, idx_g = far.voxelize(pts, voxel)
        assert np.array_equal(idx_g.cpu().numpy(), idx_o)
        assert np.array_equal(ds_g.cpu().numpy().view(np.uint32), ds_o.view(np.uint32))
    mg.close()


@gpu
@settings(max_examples=30, **SET)
@given(clouds(max_n=2000), voxels, caps, st.floats(0.0, 8.0), st.tuples(st.floats(-3, 3), st.floats(-3, 3), st.floats(-3, 3)),
       clouds(max_n=500))
def test_gpu_prune_then_reinsert_equal_oracle(pts, voxel, cap, radius, centre, more):
    far = _far()
    mo, mg = oracle.Map(voxel, cap), far.Map(voxel, cap, 1 << 13)
    mo.insert(pts); mg.insert(pts)
    assert mg.prune(centre, radius) == mo.prune(centre, radius)
    assert mg.insert(more) == mo.insert(more)                      # dead keys are re-used, ids keep counting
    eg, eo = mg.export(), mo.export()
    assert np.array_equal(eg["keys"], eo["keys"]) and np.array_equal(eg["ids"], eo["ids"])
    assert np.array_equal(eg["xyz"].view(np.uint32), eo["xyz"].view(np.uint32))
    mg.close()


@gpu
@settings(max_examples=25, **SET)
@given(clouds(max_n=1500), st.sampled_from([0.5, 1.0, 2.0]), st.integers(3, 8), st.integers(2, 6))
def test_gpu_knn_valid_flags_equal_oracle(pts, voxel, cap, k):
    far = _far()
    mo, mg = oracle.Map(voxel, cap, k_cov=k), far.Map(voxel, cap, 1 << 13, k_cov=k)
    mo.insert(pts); mg.insert(pts)
    if len(pts) == 0:
        return
    cov_o, val_o = mo.knn_cov(pts)
    cov_g, val_g = mg.knn_cov(pts)
    assert np.array_equal(val_g.cpu().numpy(), val_o)
    v = val_o.astype(bool)
    if v.any():
        a, b = cov_g.cpu().numpy()[v].astype(np.float64), cov_o[v].astype(np.float64)
        assert (np.linalg.norm(a - b, axis=1) <= 1e-4 * np.linalg.norm(b, axis=1)).all()
    mg.close()
