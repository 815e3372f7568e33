/*
 * faro.cpp -- the ORACLE: plain FP64 CPU implementation of the FAR-LIO front-end hot path.
 *
 * TEST INFRASTRUCTURE ONLY.  May be imported / linked / executed only by tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs.
 * It shares nothing with paper_2606_26010_b200/ (no kernels, headers, helpers, tables).
 *
 * Written from /root/reference/PAPER.md (cited as PAPER.md:<line>) plus the readings
 * listed in DESIGN.md section "Readings of the paper" (numbered R1..R14 there).
 * Single-threaded reference semantics; an OpenMP loop over independent queries is used
 * for timing only and never changes a result (per-point terms are summed in index order).
 * Compile with -ffp-contract=off so every FP64 operation below is one rounded IEEE op.
 *
 * Parity pins: every function below is pinned by tests/test_oracle_*.py against values the
 * paper fixes, closed forms, NumPy/SciPy library routines or brute force (see DESIGN.md,
 * "Oracle pins").  Unpinned: none in this file.
 */
#include "faro.h"

#include <algorithm>
#include <cmath>
#include <cstring>
#include <limits>
#include <unordered_map>
#include <vector>

namespace {

constexpr int32_t KEY_BIAS = 1 << 20;          // 21-bit biased index per axis
constexpr uint32_t NO_ID = 0xFFFFFFFFu;

struct Pt {
    float x, y, z;
    uint32_t id;
    float cov[6];      // xx xy xz yy yz zz (regularised, Eq. 1)
    uint8_t cov_valid;
};

struct Voxel {
    std::vector<Pt> pts;   // ascending id by construction (sequential insert)
};

// ---- A1: voxel key (reading R1: floor of the IEEE fp32 quotient) -------------
inline bool key_of(float x, float y, float z, float v, int32_t k[3]) {
    if (!std::isfinite(x) || !std::isfinite(y) || !std::isfinite(z)) return false;
    const float p[3] = {x, y, z};
    for (int a = 0; a < 3; ++a) {
        float f = std::floor(p[a] / v);            // one fp32 division, then floor
        if (!(f >= -1048576.0f && f < 1048576.0f)) return false;
        k[a] = (int32_t)f;
    }
    return true;
}

inline uint64_t pack(const int32_t k[3]) {
    return ((uint64_t)(uint32_t)(k[0] + KEY_BIAS) << 42) | ((uint64_t)(uint32_t)(k[1] + KEY_BIAS) << 21) |
           (uint64_t)(uint32_t)(k[2] + KEY_BIAS);
}

inline void unpack(uint64_t key, int32_t k[3]) {
    k[0] = (int32_t)((key >> 42) & 0x1FFFFF) - KEY_BIAS;
    k[1] = (int32_t)((key >> 21) & 0x1FFFFF) - KEY_BIAS;
    k[2] = (int32_t)(key & 0x1FFFFF) - KEY_BIAS;
}

inline bool in_range(int32_t k) { return k >= -KEY_BIAS && k < KEY_BIAS; }

// ---- A4: rigid transform in FP64, fixed operation order, rounded once to fp32 (reading R4) -
inline void transform_pt(const faro_pose_t& T, const float* s, float out[3]) {
    const double x = s[0], y = s[1], z = s[2];
    for (int r = 0; r < 3; ++r) {
        double acc = T.R[3 * r + 0] * x + T.R[3 * r + 1] * y;   // (R0*x + R1*y)
        acc = acc + T.R[3 * r + 2] * z;                          //  + R2*z
        acc = acc + T.t[r];                                      //  + t
        out[r] = (float)acc;
    }
}

// ---- small dense algebra written out by hand ---------------------------------------------
inline void sym6_to_mat(const double s[6], double m[9]) {
    m[0] = s[0]; m[1] = s[1]; m[2] = s[2];
    m[3] = s[1]; m[4] = s[3]; m[5] = s[4];
    m[6] = s[2]; m[7] = s[4]; m[8] = s[5];
}

inline bool inv3(const double a[9], double inv[9]) {
    const double c00 = a[4] * a[8] - a[5] * a[7];
    const double c01 = a[5] * a[6] - a[3] * a[8];
    const double c02 = a[3] * a[7] - a[4] * a[6];
    const double det = a[0] * c00 + a[1] * c01 + a[2] * c02;
    if (!(det != 0.0) || !std::isfinite(det)) return false;
    const double id = 1.0 / det;
    inv[0] = c00 * id;
    inv[1] = (a[2] * a[7] - a[1] * a[8]) * id;
    inv[2] = (a[1] * a[5] - a[2] * a[4]) * id;
    inv[3] = c01 * id;
    inv[4] = (a[0] * a[8] - a[2] * a[6]) * id;
    inv[5] = (a[2] * a[3] - a[0] * a[5]) * id;
    inv[6] = c02 * id;
    inv[7] = (a[1] * a[6] - a[0] * a[7]) * id;
    inv[8] = (a[0] * a[4] - a[1] * a[3]) * id;
    return true;
}

inline void mat3_mul(const double a[9], const double b[9], double c[9]) {
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
            double s = 0.0;
            for (int k = 0; k < 3; ++k) s += a[3 * i + k] * b[3 * k + j];
            c[3 * i + j] = s;
        }
}

inline void mat3_mul_bt(const double a[9], const double b[9], double c[9]) {   // a * b^T
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
            double s = 0.0;
            for (int k = 0; k < 3; ++k) s += a[3 * i + k] * b[3 * j + k];
            c[3 * i + j] = s;
        }
}

// Eq. 1: C = Sigma_hat + eps*I ; Sigma = (C^-1 / ||C^-1||_F)^-1 = ||C^-1||_F * C
bool regularised_cov(const double mean_cov[6], double eps, double out6[6]) {
    double C[9], Ci[9];
    sym6_to_mat(mean_cov, C);
    C[0] += eps; C[4] += eps; C[8] += eps;
    if (!inv3(C, Ci)) return false;
    double fro = 0.0;
    for (int i = 0; i < 9; ++i) fro += Ci[i] * Ci[i];
    fro = std::sqrt(fro);
    out6[0] = fro * C[0]; out6[1] = fro * C[1]; out6[2] = fro * C[2];
    out6[3] = fro * C[4]; out6[4] = fro * C[5]; out6[5] = fro * C[8];
    return true;
}

// sample covariance (1/k, reading R7) of k points, about their mean
void sample_cov(const double* pts /* k*3 */, int k, double out6[6]) {
    double mu[3] = {0, 0, 0};
    for (int i = 0; i < k; ++i)
        for (int a = 0; a < 3; ++a) mu[a] += pts[3 * i + a];
    for (int a = 0; a < 3; ++a) mu[a] /= (double)k;
    double s[6] = {0, 0, 0, 0, 0, 0};
    for (int i = 0; i < k; ++i) {
        const double dx = pts[3 * i] - mu[0], dy = pts[3 * i + 1] - mu[1], dz = pts[3 * i + 2] - mu[2];
        s[0] += dx * dx; s[1] += dx * dy; s[2] += dx * dz;
        s[3] += dy * dy; s[4] += dy * dz; s[5] += dz * dz;
    }
    for (int i = 0; i < 6; ++i) out6[i] = s[i] / (double)k;
}

struct Cand {
    double d2;
    uint32_t id;
    const Pt* p;
};
inline bool cand_less(const Cand& a, const Cand& b) { return a.d2 < b.d2 || (a.d2 == b.d2 && a.id < b.id); }

}  // namespace

struct faro_map {
    float voxel;
    int32_t cap;
    int32_t k_cov;
    double cov_eps;
    uint64_t next_id;
    double min_spacing = 0.0;   // R21: > 0: a point is stored only if no point already in ITS OWN voxel is closer than this
    std::unordered_map<uint64_t, Voxel> vox;

    // A6 candidate enumeration: the query's voxel and its 26 neighbours (Fig. 3)
    template <class F>
    void for_candidates(const float* q, F&& f) const {
        int32_t k[3];
        if (!key_of(q[0], q[1], q[2], voxel, k)) return;
        for (int dx = -1; dx <= 1; ++dx)
            for (int dy = -1; dy <= 1; ++dy)
                for (int dz = -1; dz <= 1; ++dz) {
                    const int32_t n[3] = {k[0] + dx, k[1] + dy, k[2] + dz};
                    if (!in_range(n[0]) || !in_range(n[1]) || !in_range(n[2])) continue;
                    auto it = vox.find(pack(n));
                    if (it == vox.end()) continue;
                    for (const Pt& p : it->second.pts) {
                        // reading R6: exact differences, each product/sum one rounded binary64 op
                        const double ddx = (double)q[0] - (double)p.x;
                        const double ddy = (double)q[1] - (double)p.y;
                        const double ddz = (double)q[2] - (double)p.z;
                        const double d2 = (ddx * ddx + ddy * ddy) + ddz * ddz;
                        f(Cand{d2, p.id, &p});
                    }
                }
    }

    bool nearest(const float* q, Cand& best) const {
        bool have = false;
        for_candidates(q, [&](const Cand& c) {
            if (!have || cand_less(c, best)) { best = c; have = true; }
        });
        return have;
    }

    // the k nearest by (d2,id); returns false if fewer than k candidates
    bool knn(const float* q, int k, std::vector<Cand>& out) const {
        out.clear();
        for_candidates(q, [&](const Cand& c) { out.push_back(c); });
        std::sort(out.begin(), out.end(), cand_less);
        if ((int)out.size() < k) return false;
        out.resize(k);
        return true;
    }

    // A7: Eq. 1 from the k nearest stored points
    bool knn_cov(const float* q, float cov6[6]) const {
        std::vector<Cand> nb;
        if (!knn(q, k_cov, nb)) {
            cov6[0] = 1; cov6[1] = 0; cov6[2] = 0; cov6[3] = 1; cov6[4] = 0; cov6[5] = 1;
            return false;
        }
        std::vector<double> pts(3 * (size_t)k_cov);
        for (int i = 0; i < k_cov; ++i) {
            pts[3 * i] = nb[i].p->x; pts[3 * i + 1] = nb[i].p->y; pts[3 * i + 2] = nb[i].p->z;
        }
        double sc[6], reg[6];
        sample_cov(pts.data(), k_cov, sc);
        if (!regularised_cov(sc, cov_eps, reg)) {
            cov6[0] = 1; cov6[1] = 0; cov6[2] = 0; cov6[3] = 1; cov6[4] = 0; cov6[5] = 1;
            return false;
        }
        for (int i = 0; i < 6; ++i) cov6[i] = (float)reg[i];
        return true;
    }
};

struct faro_threshold {
    double sigma0, min_motion, max_range;
    double sse;
    int64_t count;
};

extern "C" {

uint64_t faro_pack_key(int32_t kx, int32_t ky, int32_t kz) {
    const int32_t k[3] = {kx, ky, kz};
    return pack(k);
}
void faro_unpack_key(uint64_t key, int32_t* k3) { unpack(key, k3); }

int faro_keys(const float* xyz, int64_t n, int stride, float voxel, uint64_t* keys, uint8_t* valid) {
    if (!xyz || n < 0 || (stride != 3 && stride != 4) || !(voxel > 0)) return FARO_ERR_ARG;
    for (int64_t i = 0; i < n; ++i) {
        int32_t k[3];
        const float* p = xyz + i * stride;
        const bool ok = key_of(p[0], p[1], p[2], voxel, k);
        valid[i] = ok ? 1 : 0;
        keys[i] = ok ? pack(k) : ~0ull;
    }
    return FARO_OK;
}

// A2: for each distinct key the lowest-index valid point, in ascending source index (reading R2)
int faro_voxelize(const float* xyz, int64_t n, int stride, float voxel, float* out_xyz, int32_t* out_index,
                  int64_t* n_out) {
    if (!xyz || n < 0 || (stride != 3 && stride != 4) || !(voxel > 0)) return FARO_ERR_ARG;
    std::unordered_map<uint64_t, int64_t> seen;
    int64_t m = 0;
    for (int64_t i = 0; i < n; ++i) {
        int32_t k[3];
        const float* p = xyz + i * stride;
        if (!key_of(p[0], p[1], p[2], voxel, k)) continue;
        if (seen.emplace(pack(k), i).second) {
            out_xyz[3 * m] = p[0]; out_xyz[3 * m + 1] = p[1]; out_xyz[3 * m + 2] = p[2];
            out_index[m] = (int32_t)i;
            ++m;
        }
    }
    *n_out = m;
    return FARO_OK;
}

faro_map_t* faro_map_create(float voxel, int32_t cap, int32_t k_cov, double cov_eps) {
    if (!(voxel > 0) || cap < 1 || k_cov < 1) return nullptr;
    faro_map* m = new faro_map();
    m->voxel = voxel; m->cap = cap; m->k_cov = k_cov; m->cov_eps = cov_eps; m->next_id = 0;
    return m;
}
void faro_map_destroy(faro_map_t* m) { delete m; }
// a deep copy (the struct's own copy constructor: configuration, id counter and every voxel's point list): bookkeeping
// for callers that replay one step on the same map several times (bench.py --impl reference); no arithmetic of the method
faro_map_t* faro_map_clone(const faro_map_t* m) { return m ? new faro_map(*m) : nullptr; }
void faro_map_set_min_spacing(faro_map_t* m, double s) { if (m) m->min_spacing = s > 0.0 ? s : 0.0; }

namespace {

// R17: N_ASMD of a voxel seen from `c`; every operation one rounded binary64 operation
int32_t asmd_cap(const int32_t k[3], float voxel, const double c[3], double n_close, double d_max, int32_t k_min,
                 int32_t cap) {
    const double v = (double)voxel;
    const double dx = ((double)k[0] + 0.5) * v - c[0];
    const double dy = ((double)k[1] + 0.5) * v - c[1];
    const double dz = ((double)k[2] + 0.5) * v - c[2];
    const double d = std::sqrt((dx * dx + dy * dy) + dz * dz);
    const double f = 1.0 - d / d_max;                      // linear decay over range
    const double x = std::floor(n_close * f + 0.5);
    int32_t lim = k_min;                                   // lower bound: the k points a covariance needs
    if (x > (double)k_min) lim = (x >= (double)cap) ? cap : (int32_t)x;
    if (lim > cap) lim = cap;
    return lim;
}

// A3/A4 (reading R3): sequential semantics, lowest id wins, ids = next_id + i.
// asmd: per-voxel limit N_ASMD instead of the fixed cap (reading R17)
int insert_points(faro_map_t* m, const float* xyz, int64_t n, int stride, const faro_pose_t* pose, bool asmd,
                  double n_close, double d_max, int compute_cov, faro_insert_stats_t* stats) {
    if (!m || !xyz || n < 0 || (stride != 3 && stride != 4)) return FARO_ERR_ARG;
    if (m->next_id + (uint64_t)n > 0xFFFFFFFFull) return FARO_ERR_RANGE;
    faro_insert_stats_t st = {n, 0, 0, 0, 0};
    const double origin[3] = {0.0, 0.0, 0.0};
    const double* centre = pose ? pose->t : origin;
    std::vector<std::pair<uint64_t, uint32_t>> added;   // (key, id) of accepted points
    for (int64_t i = 0; i < n; ++i) {
        const float* s = xyz + i * stride;
        const uint32_t id = (uint32_t)(m->next_id + (uint64_t)i);
        float p[3] = {s[0], s[1], s[2]};
        if (!std::isfinite(s[0]) || !std::isfinite(s[1]) || !std::isfinite(s[2])) { st.n_invalid++; continue; }
        if (pose) transform_pt(*pose, s, p);
        int32_t k[3];
        if (!key_of(p[0], p[1], p[2], m->voxel, k)) { st.n_invalid++; continue; }
        const uint64_t key = pack(k);
        auto ins = m->vox.try_emplace(key);
        if (ins.second) st.n_new_voxels++;
        Voxel& vx = ins.first->second;
        const int32_t limit = asmd ? asmd_cap(k, m->voxel, centre, n_close, d_max, m->k_cov, m->cap) : m->cap;
        bool spaced = true;
        if (m->min_spacing > 0.0) {
            // R21 ("regularly spaced ... a minimum point-to-point distance of ~65 cm" at v = 4 m, N_max = 40,
            // i.e. v / sqrt(N_max)): sequential rule, points in index order; squared distance as R6, strict <
            const double s2 = m->min_spacing * m->min_spacing;
            for (const Pt& q : vx.pts) {
                const double dx = (double)p[0] - (double)q.x, dy = (double)p[1] - (double)q.y, dz = (double)p[2] - (double)q.z;
                const double d2 = (dx * dx + dy * dy) + dz * dz;
                if (d2 < s2) { spaced = false; break; }
            }
        }
        if ((int32_t)vx.pts.size() < limit && spaced) {
            Pt pt{p[0], p[1], p[2], id, {1, 0, 0, 1, 0, 1}, 0};
            vx.pts.push_back(pt);
            st.n_accepted++;
            if (compute_cov) added.emplace_back(key, id);
        }
    }
    m->next_id += (uint64_t)n;
    // "we recompute the covariances of the added points" -- against the map AFTER the insert
    for (auto& a : added) {
        Voxel& vx = m->vox[a.first];
        for (Pt& pt : vx.pts)
            if (pt.id == a.second) {
                const float q[3] = {pt.x, pt.y, pt.z};
                float c[6];
                pt.cov_valid = m->knn_cov(q, c) ? 1 : 0;
                std::memcpy(pt.cov, c, sizeof(c));
            }
    }
    if (stats) *stats = st;
    return FARO_OK;
}

}  // namespace

int faro_map_insert(faro_map_t* m, const float* xyz, int64_t n, int stride, const faro_pose_t* pose,
                    int compute_cov, faro_insert_stats_t* stats) {
    return insert_points(m, xyz, n, stride, pose, false, 0.0, 1.0, compute_cov, stats);
}

// SURVEY 8(f)-1, reading R17
int faro_map_insert_asmd(faro_map_t* m, const float* xyz, int64_t n, int stride, const faro_pose_t* pose,
                         double n_close, double d_max, int compute_cov, faro_insert_stats_t* stats) {
    if (!(d_max > 0.0) || !(n_close >= 0.0)) return FARO_ERR_ARG;
    return insert_points(m, xyz, n, stride, pose, true, n_close, d_max, compute_cov, stats);
}

int32_t faro_asmd_cap(const int32_t k3[3], float voxel, const double center[3], double n_close, double d_max,
                      int32_t k_min, int32_t cap) {
    return asmd_cap(k3, voxel, center, n_close, d_max, k_min, cap);
}

// PAPER.md:109 "the average amount of points per voxel in a close range of the current scan"
int faro_asmd_density(const faro_map_t* local, const double center[3], double r_close, double* n_close,
                      int64_t* n_voxels_close) {
    if (!local || !center || !n_close) return FARO_ERR_ARG;
    const double v = (double)local->voxel;
    const double r2 = r_close * r_close;
    int64_t nv = 0, np = 0;
    for (const auto& kv : local->vox) {
        if (kv.second.pts.empty()) continue;
        int32_t k[3];
        unpack(kv.first, k);
        const double dx = ((double)k[0] + 0.5) * v - center[0];
        const double dy = ((double)k[1] + 0.5) * v - center[1];
        const double dz = ((double)k[2] + 0.5) * v - center[2];
        const double d2 = (dx * dx + dy * dy) + dz * dz;
        if (d2 <= r2) { nv++; np += (int64_t)kv.second.pts.size(); }
    }
    *n_close = nv > 0 ? (double)np / (double)nv : (double)local->cap;
    if (n_voxels_close) *n_voxels_close = nv;
    return FARO_OK;
}

// A5 (reading R5): remove voxel iff squared centre distance > r*r (strict)
int faro_map_prune(faro_map_t* m, const double center[3], double radius, faro_prune_stats_t* stats) {
    if (!m || !center) return FARO_ERR_ARG;
    faro_prune_stats_t st = {0, 0, 0, 0};
    const double v = (double)m->voxel;
    const double r2 = radius * radius;
    for (auto it = m->vox.begin(); it != m->vox.end();) {
        int32_t k[3];
        unpack(it->first, k);
        const double dx = ((double)k[0] + 0.5) * v - center[0];
        const double dy = ((double)k[1] + 0.5) * v - center[1];
        const double dz = ((double)k[2] + 0.5) * v - center[2];
        const double d2 = (dx * dx + dy * dy) + dz * dz;
        if (d2 > r2) {
            st.n_voxels_removed++;
            st.n_points_removed += (int64_t)it->second.pts.size();
            it = m->vox.erase(it);
        } else {
            st.n_voxels_left++;
            st.n_points_left += (int64_t)it->second.pts.size();
            ++it;
        }
    }
    if (stats) *stats = st;
    return FARO_OK;
}

// R22: ids are this build's construct (the paper has none).  Renumbering subtracts the smallest stored id from
// every stored id and from the id counter: order, contents and every (d2, id) comparison are unchanged.  An empty map
// restarts at 0.
int faro_map_renumber(faro_map_t* m, uint64_t* subtracted) {
    if (!m) return FARO_ERR_ARG;
    uint64_t mn = m->next_id;
    for (auto& kv : m->vox)
        for (const Pt& p : kv.second.pts) mn = std::min<uint64_t>(mn, p.id);
    for (auto& kv : m->vox)
        for (Pt& p : kv.second.pts) p.id -= (uint32_t)mn;
    m->next_id -= mn;
    if (subtracted) *subtracted = mn;
    return FARO_OK;
}

int faro_map_size(const faro_map_t* m, int64_t* n_voxels, int64_t* n_points, uint64_t* next_id) {
    if (!m) return FARO_ERR_ARG;
    int64_t np = 0;
    for (auto& kv : m->vox) np += (int64_t)kv.second.pts.size();
    if (n_voxels) *n_voxels = (int64_t)m->vox.size();
    if (n_points) *n_points = np;
    if (next_id) *next_id = m->next_id;
    return FARO_OK;
}

int faro_map_export(const faro_map_t* m, uint64_t* keys, int32_t* counts, float* points4, float* cov6,
                    uint8_t* cov_valid) {
    if (!m || !keys || !counts) return FARO_ERR_ARG;
    std::vector<uint64_t> ks;
    ks.reserve(m->vox.size());
    for (auto& kv : m->vox) ks.push_back(kv.first);
    std::sort(ks.begin(), ks.end());
    const size_t cap = (size_t)m->cap;
    for (size_t v = 0; v < ks.size(); ++v) {
        const Voxel& vx = m->vox.at(ks[v]);
        keys[v] = ks[v];
        counts[v] = (int32_t)vx.pts.size();
        for (size_t j = 0; j < cap; ++j) {
            const bool have = j < vx.pts.size();
            if (points4) {
                float* o = points4 + (v * cap + j) * 4;
                uint32_t idbits = have ? vx.pts[j].id : NO_ID;
                o[0] = have ? vx.pts[j].x : 0.f;
                o[1] = have ? vx.pts[j].y : 0.f;
                o[2] = have ? vx.pts[j].z : 0.f;
                std::memcpy(o + 3, &idbits, 4);
            }
            if (cov6) {
                float* c = cov6 + (v * cap + j) * 6;
                for (int a = 0; a < 6; ++a) c[a] = have ? vx.pts[j].cov[a] : 0.f;
            }
            if (cov_valid) cov_valid[v * cap + j] = have ? vx.pts[j].cov_valid : 0;
        }
    }
    return FARO_OK;
}

int faro_map_nn(const faro_map_t* m, const float* q, int64_t n, int stride, uint32_t* id, float* d2, int nthreads) {
    if (!m || !q || n < 0 || (stride != 3 && stride != 4)) return FARO_ERR_ARG;
    if (nthreads < 1) nthreads = 1;
#pragma omp parallel for num_threads(nthreads) schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        Cand best;
        if (m->nearest(q + i * stride, best)) {
            id[i] = best.id;
            d2[i] = (float)best.d2;
        } else {
            id[i] = NO_ID;
            d2[i] = std::numeric_limits<float>::infinity();
        }
    }
    return FARO_OK;
}

// Pin helper: scans ALL stored points and applies the key-adjacency filter explicitly.
int faro_map_nn_brute(const faro_map_t* m, const float* q, int64_t n, int stride, uint32_t* id, float* d2) {
    if (!m || !q || n < 0 || (stride != 3 && stride != 4)) return FARO_ERR_ARG;
    for (int64_t i = 0; i < n; ++i) {
        const float* qq = q + i * stride;
        id[i] = NO_ID;
        d2[i] = std::numeric_limits<float>::infinity();
        int32_t kq[3];
        if (!key_of(qq[0], qq[1], qq[2], m->voxel, kq)) continue;
        double best = std::numeric_limits<double>::infinity();
        uint32_t bid = NO_ID;
        for (auto& kv : m->vox) {
            int32_t kp[3];
            unpack(kv.first, kp);
            if (std::abs(kp[0] - kq[0]) > 1 || std::abs(kp[1] - kq[1]) > 1 || std::abs(kp[2] - kq[2]) > 1) continue;
            for (const Pt& p : kv.second.pts) {
                const double dx = (double)qq[0] - (double)p.x, dy = (double)qq[1] - (double)p.y,
                             dz = (double)qq[2] - (double)p.z;
                const double d = (dx * dx + dy * dy) + dz * dz;
                if (d < best || (d == best && p.id < bid)) { best = d; bid = p.id; }
            }
        }
        if (bid != NO_ID) { id[i] = bid; d2[i] = (float)best; }
    }
    return FARO_OK;
}

int faro_map_knn(const faro_map_t* m, const float* q, int64_t n, int stride, int32_t k, uint32_t* ids, double* d2) {
    if (!m || !q || n < 0 || k < 1) return FARO_ERR_ARG;
    std::vector<Cand> nb;
    for (int64_t i = 0; i < n; ++i) {
        nb.clear();
        m->for_candidates(q + i * stride, [&](const Cand& c) { nb.push_back(c); });
        std::sort(nb.begin(), nb.end(), cand_less);
        for (int32_t j = 0; j < k; ++j) {
            const bool have = j < (int32_t)nb.size();
            ids[i * k + j] = have ? nb[j].id : NO_ID;
            d2[i * k + j] = have ? nb[j].d2 : std::numeric_limits<double>::infinity();
        }
    }
    return FARO_OK;
}

int faro_map_knn_cov(const faro_map_t* m, const float* q, int64_t n, int stride, float* cov6, uint8_t* valid,
                     int nthreads) {
    if (!m || !q || n < 0 || (stride != 3 && stride != 4)) return FARO_ERR_ARG;
    if (nthreads < 1) nthreads = 1;
#pragma omp parallel for num_threads(nthreads) schedule(static)
    for (int64_t i = 0; i < n; ++i) valid[i] = m->knn_cov(q + i * stride, cov6 + 6 * i) ? 1 : 0;
    return FARO_OK;
}

int faro_cov_from_points(const float* pts, int32_t k, int stride, double eps, double* cov6_out) {
    if (!pts || k < 1) return FARO_ERR_ARG;
    std::vector<double> p(3 * (size_t)k);
    for (int i = 0; i < k; ++i)
        for (int a = 0; a < 3; ++a) p[3 * i + a] = pts[i * stride + a];
    double sc[6];
    sample_cov(p.data(), k, sc);
    return regularised_cov(sc, eps, cov6_out) ? FARO_OK : FARO_ERR_DEGENERATE;
}

void faro_gicp_default_options(faro_gicp_options_t* o) {
    o->kernel = FARO_KERNEL_CAUCHY;
    o->conv_eps = 5e-3;
    o->tau_mult = 3.0;
    o->kappa_div = 3.0;
}

// reading R9: IRLS weight of the robust kernel on e = sqrt(d^T M d)
double faro_robust_weight(int kernel, double e2, double kappa) {
    switch (kernel) {
        case FARO_KERNEL_CAUCHY: return 1.0 / (1.0 + e2 / (kappa * kappa));          // Eq. 5
        case FARO_KERNEL_GEMAN_MCCLURE: { const double s = kappa + e2; return (kappa * kappa) / (s * s); }
        default: return 1.0;
    }
}

// SE(3) exponential, delta = (rho, phi), translation first (reading R12)
void faro_se3_exp(const double d[6], faro_pose_t* out) {
    const double rho[3] = {d[0], d[1], d[2]};
    const double phi[3] = {d[3], d[4], d[5]};
    const double th2 = phi[0] * phi[0] + phi[1] * phi[1] + phi[2] * phi[2];
    const double th = std::sqrt(th2);
    double A, B, C;
    if (th < 1e-8) {
        A = 1.0 - th2 / 6.0;
        B = 0.5 - th2 / 24.0;
        C = 1.0 / 6.0 - th2 / 120.0;
    } else {
        A = std::sin(th) / th;
        B = (1.0 - std::cos(th)) / th2;
        C = (th - std::sin(th)) / (th2 * th);
    }
    const double K[9] = {0, -phi[2], phi[1], phi[2], 0, -phi[0], -phi[1], phi[0], 0};
    double K2[9];
    mat3_mul(K, K, K2);
    double V[9];
    for (int i = 0; i < 9; ++i) {
        const double I = (i % 4 == 0) ? 1.0 : 0.0;
        out->R[i] = I + A * K[i] + B * K2[i];
        V[i] = I + B * K[i] + C * K2[i];
    }
    for (int r = 0; r < 3; ++r) out->t[r] = V[3 * r] * rho[0] + V[3 * r + 1] * rho[1] + V[3 * r + 2] * rho[2];
}

namespace {

struct Corr {
    bool used;
    double p[3], r[3], M[9], w, e2;
    uint32_t id;
};

// A8 + A9 for ONE source point (Eq. 2-5)
Corr correspond(const faro_map& m, const float* s, const float* cov_s, bool valid_s, const faro_pose_t& T,
                double sigma, const faro_gicp_options_t& o) {
    Corr c{};
    c.used = false;
    c.id = NO_ID;
    if (!std::isfinite(s[0]) || !std::isfinite(s[1]) || !std::isfinite(s[2])) return c;
    float pf[3];
    transform_pt(T, s, pf);                                   // Eq. 2 / accumulated pose (reading R11)
    Cand best;
    if (!m.nearest(pf, best)) return c;                       // kNN-search, k=1
    const double tau = o.tau_mult * sigma;
    if (best.d2 > tau * tau) return c;                        // adaptive threshold gate
    c.id = best.id;
    for (int a = 0; a < 3; ++a) c.p[a] = pf[a];
    c.r[0] = best.p->x; c.r[1] = best.p->y; c.r[2] = best.p->z;
    const double d[3] = {c.r[0] - c.p[0], c.r[1] - c.p[1], c.r[2] - c.p[2]};   // Eq. 3
    bool full = valid_s && best.p->cov_valid;
    if (full) {
        // M = (Sigma_r + R Sigma_s R^T)^-1   (Eq. 4)
        double Ss[9], RS[9], RSRt[9], Sr[9], S[9];
        const double cs[6] = {cov_s[0], cov_s[1], cov_s[2], cov_s[3], cov_s[4], cov_s[5]};
        const double cr[6] = {best.p->cov[0], best.p->cov[1], best.p->cov[2], best.p->cov[3], best.p->cov[4],
                              best.p->cov[5]};
        sym6_to_mat(cs, Ss);
        sym6_to_mat(cr, Sr);
        mat3_mul(T.R, Ss, RS);
        mat3_mul_bt(RS, T.R, RSRt);
        for (int i = 0; i < 9; ++i) S[i] = Sr[i] + RSRt[i];
        if (!inv3(S, c.M)) full = false;
    }
    if (!full) {   // sparsity-aware fallback: Sigma_r = I, Sigma_s = 0
        for (int i = 0; i < 9; ++i) c.M[i] = (i % 4 == 0) ? 1.0 : 0.0;
    }
    double Md[3];
    for (int r = 0; r < 3; ++r) Md[r] = c.M[3 * r] * d[0] + c.M[3 * r + 1] * d[1] + c.M[3 * r + 2] * d[2];
    c.e2 = d[0] * Md[0] + d[1] * Md[1] + d[2] * Md[2];
    c.w = faro_robust_weight(o.kernel, c.e2, sigma / o.kappa_div);
    c.used = true;
    return c;
}

// accumulate w J^T M J and w J^T M d with J = [ -I | [p]x ]  (reading R12)
void accumulate(const Corr& c, double H[36], double b[6]) {
    const double px = c.p[0], py = c.p[1], pz = c.p[2];
    const double J[18] = {-1, 0, 0, 0, -pz, py,
                          0, -1, 0, pz, 0, -px,
                          0, 0, -1, -py, px, 0};
    const double d[3] = {c.r[0] - c.p[0], c.r[1] - c.p[1], c.r[2] - c.p[2]};
    double MJ[18];   // 3x6
    for (int r = 0; r < 3; ++r)
        for (int k = 0; k < 6; ++k)
            MJ[6 * r + k] = c.M[3 * r] * J[k] + c.M[3 * r + 1] * J[6 + k] + c.M[3 * r + 2] * J[12 + k];
    double Md[3];
    for (int r = 0; r < 3; ++r) Md[r] = c.M[3 * r] * d[0] + c.M[3 * r + 1] * d[1] + c.M[3 * r + 2] * d[2];
    for (int a = 0; a < 6; ++a) {
        for (int k = 0; k < 6; ++k)
            H[6 * a + k] += c.w * (J[a] * MJ[k] + J[6 + a] * MJ[6 + k] + J[12 + a] * MJ[12 + k]);
        b[a] += c.w * (J[a] * Md[0] + J[6 + a] * Md[1] + J[12 + a] * Md[2]);
    }
}

// 6x6 Cholesky solve of H x = rhs; false if H is not positive definite
bool chol_solve6(const double H[36], const double rhs[6], double x[6]) {
    double L[36] = {0};
    for (int i = 0; i < 6; ++i)
        for (int j = 0; j <= i; ++j) {
            double s = H[6 * i + j];
            for (int k = 0; k < j; ++k) s -= L[6 * i + k] * L[6 * j + k];
            if (i == j) {
                if (!(s > 0.0) || !std::isfinite(s)) return false;
                L[6 * i + i] = std::sqrt(s);
            } else {
                L[6 * i + j] = s / L[6 * j + j];
            }
        }
    double y[6];
    for (int i = 0; i < 6; ++i) {
        double s = rhs[i];
        for (int k = 0; k < i; ++k) s -= L[6 * i + k] * y[k];
        y[i] = s / L[6 * i + i];
    }
    for (int i = 5; i >= 0; --i) {
        double s = y[i];
        for (int k = i + 1; k < 6; ++k) s -= L[6 * k + i] * x[k];
        x[i] = s / L[6 * i + i];
    }
    return true;
}

void linearise(const faro_map& m, const float* scan, const float* cov6, const uint8_t* valid, int64_t n, int stride,
               const faro_pose_t& T, double sigma, const faro_gicp_options_t& o, faro_gicp_result_t& out,
               int nthreads) {
    std::vector<Corr> cs((size_t)n);
#pragma omp parallel for num_threads(nthreads) schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        static const float ident[6] = {1, 0, 0, 1, 0, 1};
        const bool vs = (cov6 && valid) ? valid[i] != 0 : false;
        cs[(size_t)i] = correspond(m, scan + i * stride, cov6 ? cov6 + 6 * i : ident, vs, T, sigma, o);
    }
    std::memset(out.H, 0, sizeof(out.H));
    std::memset(out.b, 0, sizeof(out.b));
    out.chi2 = 0.0;
    out.n_inliers = 0;
    for (int64_t i = 0; i < n; ++i) {          // index order: result independent of nthreads
        const Corr& c = cs[(size_t)i];
        if (!c.used) continue;
        accumulate(c, out.H, out.b);
        out.chi2 += c.w * c.e2;
        out.n_inliers++;
    }
}

}  // namespace

int faro_gicp_correspondences(const faro_map_t* m, const float* scan, const float* cov6, const uint8_t* valid,
                              int64_t n, int stride, const faro_pose_t* pose, double sigma,
                              const faro_gicp_options_t* opts, uint8_t* used, double* p3, double* r3, double* M9,
                              double* w, uint32_t* id) {
    if (!m || !scan || !pose) return FARO_ERR_ARG;
    faro_gicp_options_t o;
    if (opts) o = *opts; else faro_gicp_default_options(&o);
    static const float ident[6] = {1, 0, 0, 1, 0, 1};
    for (int64_t i = 0; i < n; ++i) {
        const bool vs = (cov6 && valid) ? valid[i] != 0 : false;
        Corr c = correspond(*m, scan + i * stride, cov6 ? cov6 + 6 * i : ident, vs, *pose, sigma, o);
        used[i] = c.used;
        for (int a = 0; a < 3; ++a) { p3[3 * i + a] = c.p[a]; r3[3 * i + a] = c.r[a]; }
        for (int a = 0; a < 9; ++a) M9[9 * i + a] = c.M[a];
        w[i] = c.w;
        id[i] = c.id;
    }
    return FARO_OK;
}

int faro_gicp_linearize(const faro_map_t* m, const float* scan, const float* cov6, const uint8_t* valid, int64_t n,
                        int stride, const faro_pose_t* pose, double sigma, const faro_gicp_options_t* opts,
                        faro_gicp_result_t* out, int nthreads) {
    if (!m || !scan || !pose || !out || n < 0 || (stride != 3 && stride != 4)) return FARO_ERR_ARG;
    faro_gicp_options_t o;
    if (opts) o = *opts; else faro_gicp_default_options(&o);
    if (nthreads < 1) nthreads = 1;
    linearise(*m, scan, cov6, valid, n, stride, *pose, sigma, o, *out, nthreads);
    out->pose = *pose;
    out->iters = 1;
    out->converged = 0;
    out->status = FARO_OK;
    return FARO_OK;
}

// Gauss-Newton loop: linearise, solve H delta = -b, T <- Exp(delta) T
int faro_gicp_register(const faro_map_t* m, const float* scan, const float* cov6, const uint8_t* valid, int64_t n,
                       int stride, const faro_pose_t* init, double sigma, int max_iters,
                       const faro_gicp_options_t* opts, faro_gicp_result_t* out, int nthreads) {
    if (!m || !scan || !init || !out || n < 0 || (stride != 3 && stride != 4) || max_iters < 1) return FARO_ERR_ARG;
    faro_gicp_options_t o;
    if (opts) o = *opts; else faro_gicp_default_options(&o);
    if (nthreads < 1) nthreads = 1;
    faro_pose_t T = *init;
    out->converged = 0;
    out->status = FARO_OK;
    out->iters = 0;
    for (int it = 0; it < max_iters; ++it) {
        linearise(*m, scan, cov6, valid, n, stride, T, sigma, o, *out, nthreads);
        out->iters = it + 1;
        double rhs[6], delta[6];
        for (int a = 0; a < 6; ++a) rhs[a] = -out->b[a];
        if (out->n_inliers < 6 || !chol_solve6(out->H, rhs, delta)) {
            out->status = FARO_ERR_DEGENERATE;
            T = *init;
            break;
        }
        faro_pose_t E, Tn;
        faro_se3_exp(delta, &E);
        mat3_mul(E.R, T.R, Tn.R);                                   // T <- Exp(delta) * T   (Eq. 6)
        for (int r = 0; r < 3; ++r)
            Tn.t[r] = (E.R[3 * r] * T.t[0] + E.R[3 * r + 1] * T.t[1] + E.R[3 * r + 2] * T.t[2]) + E.t[r];
        T = Tn;
        double nrm = 0.0;
        for (int a = 0; a < 6; ++a) nrm += delta[a] * delta[a];
        if (std::sqrt(nrm) <= o.conv_eps) {                          // PAPER.md:100, reading R13
            out->converged = 1;
            break;
        }
    }
    out->pose = T;
    return FARO_OK;
}

// ---- adaptive threshold (reading R10) ------------------------------------------
faro_threshold_t* faro_threshold_create(double sigma0, double min_motion, double max_range) {
    faro_threshold* t = new faro_threshold{sigma0, min_motion, max_range, 0.0, 0};
    return t;
}
void faro_threshold_destroy(faro_threshold_t* t) { delete t; }

void faro_threshold_update(faro_threshold_t* t, const faro_pose_t* pred, const faro_pose_t* reg) {
    // deviation dT = pred^-1 * reg
    double Rt[9], dR[9];
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) Rt[3 * i + j] = pred->R[3 * j + i];
    mat3_mul(Rt, reg->R, dR);
    const double dtw[3] = {reg->t[0] - pred->t[0], reg->t[1] - pred->t[1], reg->t[2] - pred->t[2]};
    double dt[3];
    for (int r = 0; r < 3; ++r) dt[r] = Rt[3 * r] * dtw[0] + Rt[3 * r + 1] * dtw[1] + Rt[3 * r + 2] * dtw[2];
    double c = 0.5 * ((dR[0] + dR[4] + dR[8]) - 1.0);
    c = std::min(1.0, std::max(-1.0, c));
    const double theta = std::acos(c);
    const double delta = std::sqrt(dt[0] * dt[0] + dt[1] * dt[1] + dt[2] * dt[2]) +
                         2.0 * t->max_range * std::sin(0.5 * theta);
    if (delta > t->min_motion) {
        t->sse += delta * delta;
        t->count++;
    }
}

double faro_threshold_sigma(const faro_threshold_t* t) {
    if (t->count == 0) return t->sigma0;
    return std::sqrt(t->sse / (double)t->count);
}


// ---- motion undistortion (readings R15/R16) -----------------------------------
// R15: ordinary least squares line x(t) = a + b (t - t_ref) per twist component
int faro_motion_fit(const double* times, const double* vel6, int32_t m, double t_ref, faro_motion_t* out) {
    if (!times || !vel6 || !out || m < 1) return FARO_ERR_ARG;
    double sbar = 0.0;
    for (int32_t j = 0; j < m; ++j) sbar += times[j] - t_ref;
    sbar /= (double)m;
    double sxx = 0.0;
    for (int32_t j = 0; j < m; ++j) { const double ds = (times[j] - t_ref) - sbar; sxx += ds * ds; }
    for (int c = 0; c < 6; ++c) {
        double xbar = 0.0;
        for (int32_t j = 0; j < m; ++j) xbar += vel6[6 * j + c];
        xbar /= (double)m;
        double sxy = 0.0;
        for (int32_t j = 0; j < m; ++j) sxy += ((times[j] - t_ref) - sbar) * (vel6[6 * j + c] - xbar);
        const double slope = sxx > 0.0 ? sxy / sxx : 0.0;
        out->b[c] = slope;
        out->a[c] = xbar - slope * sbar;          // value of the line at t = t_ref
    }
    return FARO_OK;
}

// R16: Magnus expansion (to second order) of the linear twist between the point's time and t_ref.
// dG/dt = G [xi(t)]^ (body twist), xi(t) = a + b (t - t_ref), Delta = t_ref - t_i:
//   Omega_1 = int xi = a Delta - b Delta^2 / 2
//   Omega_2 = +(1/2) int int [xi(s1), xi(s2)] ds2 ds1 (sign of the right-multiplied ODE) = [a, b] Delta^3 / 12
//   with the se(3) bracket [(v1,w1),(v2,w2)] = (w1 x v2 - w2 x v1, w1 x w2);  G(t_i)^-1 G(t_ref) = Exp(Omega_1 + Omega_2)
// and the point moves by the inverse: out = fl32(Exp(-(Omega_1 + Omega_2)) p).
int faro_undistort(const float* xyz, const float* time, int64_t n, int stride, double dt_ref,
                   const faro_motion_t* motion, float* out_xyz) {
    if ((!xyz && n > 0) || (!time && n > 0) || !motion || (!out_xyz && n > 0) || n < 0 || (stride != 3 && stride != 4))
        return FARO_ERR_ARG;
    const double* a = motion->a;
    const double* b = motion->b;
    const double* va = a;      const double* wa = a + 3;
    const double* vb = b;      const double* wb = b + 3;
    double br[6];              // [a, b]
    br[0] = (wa[1] * vb[2] - wa[2] * vb[1]) - (wb[1] * va[2] - wb[2] * va[1]);
    br[1] = (wa[2] * vb[0] - wa[0] * vb[2]) - (wb[2] * va[0] - wb[0] * va[2]);
    br[2] = (wa[0] * vb[1] - wa[1] * vb[0]) - (wb[0] * va[1] - wb[1] * va[0]);
    br[3] = wa[1] * wb[2] - wa[2] * wb[1];
    br[4] = wa[2] * wb[0] - wa[0] * wb[2];
    br[5] = wa[0] * wb[1] - wa[1] * wb[0];
    for (int64_t i = 0; i < n; ++i) {
        const float* s = xyz + i * stride;
        float* o = out_xyz + 3 * i;
        if (!std::isfinite(s[0]) || !std::isfinite(s[1]) || !std::isfinite(s[2]) || !std::isfinite(time[i])) {
            o[0] = s[0]; o[1] = s[1]; o[2] = s[2];
            continue;
        }
        const double D = dt_ref - (double)time[i];
        const double h = 0.5 * (D * D);
        const double g = (D * D) * D / 12.0;
        double neg_omega[6];
        for (int c = 0; c < 6; ++c) neg_omega[c] = -((a[c] * D - b[c] * h) + br[c] * g);
        faro_pose_t E;
        faro_se3_exp(neg_omega, &E);
        transform_pt(E, s, o);
    }
    return FARO_OK;
}

}  // extern "C"
