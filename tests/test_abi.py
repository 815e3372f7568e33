"""CPU-only checks of the boundary: libfar.so builds for sm_100a, loads without a GPU and exports every
function include/far.h declares; struct layouts of the binding match the header's; host-only helpers work."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "far.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = set(re.findall(r"\b(far_[a-z0-9_]+)\s*\(", src))
    return sorted(names)


def test_header_declares_the_north_star_calls():
    names = _declared_functions()
    for required in ("far_map_create", "far_map_insert", "far_map_prune", "far_voxelize", "far_gicp_register",
                     "far_map_nn", "far_map_knn_cov", "far_gicp_linearize", "far_map_export"):
        assert required in names


def test_library_builds_loads_and_exports_every_declared_symbol():
    import paper_2606_26010_b200 as far
    L = far.lib()
    assert os.path.exists(far.LIB_PATH)
    for name in _declared_functions():
        assert hasattr(L, name), f"libfar.so does not export {name}"
    # the binding gives a prototype to every declared function
    assert set(L._far_symbols) == set(_declared_functions())
    assert L.far_strerror(0) == b"ok"
    assert L.far_strerror(5).startswith(b"degenerate")


def test_library_is_sm100a_with_no_other_arch():
    import subprocess
    import paper_2606_26010_b200 as far
    far.lib()
    out = subprocess.run(["/usr/local/cuda/bin/cuobjdump", "-lelf", far.LIB_PATH], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_(\d+a?)", out))
    assert archs == {"100a"}, archs


def test_struct_sizes_match_header_layout():
    import paper_2606_26010_b200 as far
    assert C.sizeof(far.Pose) == 96
    assert C.sizeof(far.GicpOptions) == 32
    assert C.sizeof(far.GicpResult) == 96 + 36 * 8 + 6 * 8 + 8 + 16
    assert C.sizeof(far.MapConfig) == 64
    assert C.sizeof(far.FrontendConfig) == 64 + 8 + 8 + 8 + 8 + 32 + 8 + 8 + 8 + 8
    assert C.sizeof(far.Motion) == 96


def test_default_options_are_the_papers():
    import paper_2606_26010_b200 as far
    o = far.GicpOptions()
    far.lib().far_gicp_default_options(C.byref(o))
    assert (o.kernel, o.conv_eps, o.tau_mult, o.kappa_div) == (far.KERNEL_CAUCHY, 5e-3, 3.0, 3.0)


def test_threshold_helper_matches_oracle_and_closed_form():
    import oracle
    import paper_2606_26010_b200 as far
    from far_scenes import pose_from_rpy_t, pose_identity
    rng = np.random.default_rng(5)
    a, b = far.AdaptiveThreshold(2.0, 0.1, 100.0), oracle.AdaptiveThreshold(2.0, 0.1, 100.0)
    assert a.sigma() == 2.0
    pred = pose_identity()
    # closed form after one recorded deviation: |dt| + 2 r sin(theta/2)
    reg = pose_from_rpy_t(0, 0, 0.01, [0.3, 0.0, 0.0])
    a.update(pred, reg); b.update(pred, reg)
    assert a.sigma() == pytest.approx(0.3 + 2 * 100.0 * np.sin(0.005), rel=1e-12)
    assert a.sigma() == pytest.approx(b.sigma(), rel=1e-12)
    for _ in range(20):
        pred = pose_from_rpy_t(*rng.normal(0, 0.3, 3), rng.normal(0, 5, 3))
        reg = pose_from_rpy_t(*rng.normal(0, 0.3, 3), rng.normal(0, 5, 3))
        a.update(pred, reg); b.update(pred, reg)
        assert a.sigma() == pytest.approx(b.sigma(), rel=1e-10)
    # below min_motion: unchanged
    s0 = a.sigma()
    a.update(pose_identity(), pose_from_rpy_t(0, 0, 0, [0.01, 0, 0]))
    assert a.sigma() == s0


def test_motion_fit_helper_matches_oracle_and_polyfit():
    """far_motion_fit is host-only FP64 boundary logic (R15): same line as the oracle's and NumPy's polyfit"""
    import oracle
    import paper_2606_26010_b200 as far
    rng = np.random.default_rng(7)
    t_ref = 50.0
    times = t_ref - np.sort(rng.uniform(0, 0.25, 20))[::-1]
    vel = rng.normal(0, 0.5, (20, 6)) + np.array([65.0, 0, 0, 0, 0, 0.3]) + np.outer(times - t_ref, [3, 0, 0, 0, 0, 1.0])
    a, b = far.motion_fit(times, vel, t_ref)
    ao, bo = oracle.motion_fit(times, vel, t_ref)
    assert np.allclose(a, ao, rtol=1e-12, atol=1e-12) and np.allclose(b, bo, rtol=1e-10, atol=1e-10)
    for c in range(6):
        slope, icpt = np.polyfit(times - t_ref, vel[:, c], 1)
        assert abs(b[c] - slope) < 1e-8 and abs(a[c] - icpt) < 1e-9
    a, b = far.motion_fit(times[:1], vel[:1], t_ref)
    assert np.array_equal(b, np.zeros(6)) and np.allclose(a, vel[0])


def test_compute_calls_fail_loudly_without_a_gpu():
    import torch
    import paper_2606_26010_b200 as far
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        far.Map(0.5, 20, 1024)


def test_insert_calls_reject_a_null_map_instead_of_dereferencing_it():
    """FAR_ERR_ARG = "null pointer, bad stride/size/config" (far.h): the four insert entry points check the handle before
    they read anything through it (host-side argument check only: no GPU needed, nothing is enqueued)."""
    import paper_2606_26010_b200 as far
    L = far.lib()
    dummy = (C.c_double * 16)()                      # stands in for the non-null pose / n_close pointers; never read
    d = C.cast(dummy, C.c_void_p)
    assert L.far_map_insert(None, d, 4, 3, None, 0, None, None) == far.ERR_ARG
    assert L.far_map_insert(None, None, 0, 3, None, 0, None, None) == far.ERR_ARG
    assert L.far_map_insert_dev(None, d, 4, 3, d, 0, None, None) == far.ERR_ARG
    assert L.far_map_insert_asmd(None, d, 4, 3, None, d, 50.0, 0, None, None) == far.ERR_ARG
    assert L.far_map_insert_asmd_dev(None, d, 4, 3, d, d, 50.0, 0, None, None) == far.ERR_ARG
