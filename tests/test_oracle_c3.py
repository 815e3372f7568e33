"""BASELINE.json configs[2] says "constant-velocity initial guess": T_pred = T_{t-1} (T_{t-2}^-1 T_{t-1}).

Rounds 1-2 of this repository (and the round-2 review's own replay) found that with this guess the registration drifts
out of its basin on the procedural race track after ~30 frames -- 0.18 m along-track at frame 30, 6 m at frame 41,
FAR_ERR_DEGENERATE from frame 47 -- and therefore ran the 200-frame sequence on the Sensor Fusion prior instead
(PAPER.md:76, :113).  The replay below, on the oracle alone (no GPU; seed 2, s0 = 300 m), shows what that drift really
was: an artefact of how the PREDICTION was composed, not a property of the method.  The product of three pose matrices
with a transpose standing in for the inverse multiplies any deviation of R from orthonormality from frame to frame; the
registration (T <- Exp(delta) T) preserves whatever R it is given, so the deviation is fed back and
grows geometrically (1e-11 in the bootstrap poses, 2e-8 by frame 22) until the "pose" is no rigid transform any more.
(a) With the predicted rotation projected back onto SO(3) -- a predicted pose is a rigid transform -- the literal
    constant-velocity guess is well-posed: every frame converges within a few iterations and stays within 0.2 m of
    the ground truth along the track, sigma stays at ~0.15 m.
(b) Without the projection the same loop reproduces the divergence reported earlier, together with its cause: the
    orthonormality defect of the registered pose, growing by orders of magnitude.
The 200-frame parity test and the bench leg keep the Sensor Fusion prior because it is the paper's loop,
not because the constant-velocity guess fails; the GPU parity test of the literal guess (tests/test_gpu_full_size.py)
uses the projected prediction of (a).
"""
import numpy as np
import pytest

import far_scenes as scenes
import oracle

ERR_DEGENERATE = 5


@pytest.fixture(scope="module")
def c3_frames():
    track = scenes.RaceTrack(seed=2)
    rng = np.random.default_rng(2)
    return [scenes.c3_racing_frame(track, 300.0 + 6.94 * f, rng) for f in range(51)]


def _replay(frames, project):
    v, cap, prune_r = 1.0, 20, 200.0
    mo = oracle.Map(v, cap)
    th = oracle.AdaptiveThreshold(2.0, 0.1, 200.0)
    P = []
    for f in range(2):
        mo.insert(frames[f][0], pose=frames[f][1], compute_cov=True)
        P.append(frames[f][1])
    log = {}
    for f in range(2, len(frames)):
        scan, T_gt = frames[f]
        R, t = scenes.pose_compose(P[-1], scenes.pose_compose(scenes.pose_inverse(P[-2]), P[-1]))
        if project:
            U, _, Vt = np.linalg.svd(R)
            R = U @ Vt
        pred = (R, t)
        ds, _ = oracle.voxelize(scan, v)
        lo = oracle.Map(v, cap)
        lo.insert(scan)
        cov, val = lo.knn_cov(ds, nthreads=8)
        sigma = th.sigma()
        o = mo.gicp_register(ds, cov, val, pred, sigma, 30, nthreads=8)
        T = (o["R"], o["t"])
        mo.insert(scan, pose=T, compute_cov=True)
        mo.prune(o["t"], prune_r)
        th.update(pred, T)
        P.append(T)
        log[f] = dict(status=o["status"], converged=o["converged"], iters=o["iters"], sigma=sigma,
                      along=float((T_gt[0].T @ (o["t"] - T_gt[1]))[0]),
                      ortho=float(np.abs(o["R"].T @ o["R"] - np.eye(3)).max()))
    return log


def test_c3_constant_velocity_guess_is_well_posed_when_the_prediction_is_a_rigid_transform(c3_frames):
    log = _replay(c3_frames, project=True)
    for f, r in log.items():
        assert r["status"] == 0 and r["converged"] == 1 and r["iters"] <= 12, (f, r)
        assert abs(r["along"]) < 0.2 and r["ortho"] < 1e-12, (f, r)
    assert 0.1 < log[50]["sigma"] < 0.3


def test_c3_divergence_reported_earlier_is_the_unprojected_composition_losing_orthonormality(c3_frames):
    log = _replay(c3_frames, project=False)
    for f in range(2, 30):
        assert log[f]["status"] == 0 and log[f]["converged"] == 1 and abs(log[f]["along"]) < 0.2, (f, log[f])
    # the cause: the registered "rotation" drifts away from orthonormality by orders of magnitude ...
    assert log[2]["ortho"] < 1e-9 and log[22]["ortho"] > 1e-9 and log[41]["ortho"] > 1e3 * log[22]["ortho"], \
        (log[2]["ortho"], log[22]["ortho"], log[41]["ortho"])
    # ... and the symptoms reported in rounds 1-2: along-track error, runaway threshold, no convergence, degenerate
    assert abs(log[41]["along"]) > 3.0 and log[41]["sigma"] > 100 * log[20]["sigma"], log[41]
    not_converged = [f for f in log if log[f]["status"] == 0 and not log[f]["converged"]]
    degenerate = [f for f in log if log[f]["status"] == ERR_DEGENERATE]
    assert not_converged and 38 <= not_converged[0] <= 46, not_converged
    assert degenerate and 43 <= degenerate[0] <= 50 and degenerate == list(range(degenerate[0], 51)), degenerate
