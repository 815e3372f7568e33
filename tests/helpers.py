"""NumPy/SciPy restatements used to PIN the oracle (independent of oracle/ and of the CUDA path)."""
import json
import os

import numpy as np

BIAS = 1 << 20


def load_golden(name):
    here = os.path.dirname(os.path.abspath(__file__))
    with open(os.path.join(here, "golden", name)) as f:
        return json.load(f)


def np_voxel_index(xyz, voxel):
    """floor of the IEEE fp32 quotient, as int64 (N,3)."""
    q = np.asarray(xyz, dtype=np.float32)[:, :3] / np.float32(voxel)
    assert q.dtype == np.float32
    return np.floor(q).astype(np.int64)


def np_pack(k):
    k = np.asarray(k, dtype=np.int64)
    return ((k[..., 0] + BIAS).astype(np.uint64) << np.uint64(42)) | \
           ((k[..., 1] + BIAS).astype(np.uint64) << np.uint64(21)) | (k[..., 2] + BIAS).astype(np.uint64)


def np_unpack(keys):
    keys = np.asarray(keys, dtype=np.uint64)
    m = np.uint64(0x1FFFFF)
    return np.stack([((keys >> np.uint64(42)) & m).astype(np.int64) - BIAS,
                     ((keys >> np.uint64(21)) & m).astype(np.int64) - BIAS,
                     (keys & m).astype(np.int64) - BIAS], axis=-1)


def np_capped_contents(xyz, voxel, cap, first_id=0):
    """Sequential capped insert restated with a stable argsort: dict key -> list of ids (ascending)."""
    keys = np_pack(np_voxel_index(xyz, voxel))
    order = np.argsort(keys, kind="stable")
    ks = keys[order]
    starts = np.nonzero(np.r_[True, ks[1:] != ks[:-1]])[0]
    ends = np.r_[starts[1:], len(ks)]
    return {int(ks[s]): (order[s:min(e, s + cap)] + first_id).tolist() for s, e in zip(starts, ends)}


def np_nn_bruteforce(map_xyz, map_ids, q, voxel):
    """27-voxel nearest neighbour by exhaustive search in float64 with the key-adjacency filter."""
    mk = np_voxel_index(map_xyz, voxel)
    qk = np_voxel_index(q, voxel)
    mp = np.asarray(map_xyz, dtype=np.float64)
    ids = np.full(len(q), 0xFFFFFFFF, dtype=np.uint32)
    d2o = np.full(len(q), np.inf, dtype=np.float64)
    for i in range(len(q)):
        adj = np.all(np.abs(mk - qk[i]) <= 1, axis=1)
        if not adj.any():
            continue
        d = np.asarray(q[i], dtype=np.float64) - mp[adj]
        d2 = (d[:, 0] * d[:, 0] + d[:, 1] * d[:, 1]) + d[:, 2] * d[:, 2]
        cid = np.asarray(map_ids)[adj]
        best = np.lexsort((cid, d2))[0]
        ids[i] = cid[best]
        d2o[i] = d2[best]
    return ids, d2o


def export_to_dict(exp):
    """{key: [(id, x, y, z), ...]} from an export dict (oracle or CUDA binding)."""
    out = {}
    for v in range(len(exp["keys"])):
        c = int(exp["counts"][v])
        out[int(exp["keys"][v])] = [(int(exp["ids"][v, j]),) + tuple(float(x) for x in exp["xyz"][v, j]) for j in range(c)]
    return out


def hat(v):
    return np.array([[0, -v[2], v[1]], [v[2], 0, -v[0]], [-v[1], v[0], 0]], dtype=np.float64)


def twist_matrix(delta):
    X = np.zeros((4, 4))
    X[:3, :3] = hat(delta[3:])
    X[:3, 3] = delta[:3]
    return X


def rot_angle(R):
    return float(np.arccos(np.clip(0.5 * (np.trace(R) - 1.0), -1.0, 1.0)))


def rot_sin(R):
    """sin of the rotation angle of R from its antisymmetric part.  For the tiny angles parity is about (1e-5 rad and below)
    this is the well-conditioned measure: arccos of the trace (rot_angle) turns a deviation eps of the trace -- e.g. a
    non-orthonormality of 1e-10 that both chains of a sequence share -- into an angle of sqrt(2 eps)."""
    w = np.array([R[2, 1] - R[1, 2], R[0, 2] - R[2, 0], R[1, 0] - R[0, 1]])
    return float(0.5 * np.linalg.norm(w))
