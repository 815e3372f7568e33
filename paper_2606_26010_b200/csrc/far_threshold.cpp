// far_threshold.cpp -- host-only FP64 helper: the adaptive correspondence threshold of Vizzo et al. [1]
// ("adaptive thresholding scheme from Vizzo et al.", PAPER.md:92 kappa "dynamically adjusted ...
// analogous to Vizzo et al."), as read in DESIGN.md R10.  Boundary logic, not a kernel: the hot path only
// receives the resulting sigma.
#include <algorithm>
#include <cmath>
#include <cstdint>

#include "../../include/far.h"

struct far_threshold {
    double sigma0, min_motion, max_range;
    double sum_sq;
    int64_t count;
};

extern "C" {

far_threshold_t* far_threshold_create(double sigma0, double min_motion, double max_range) {
    return new far_threshold{sigma0, min_motion, max_range, 0.0, 0};
}

void far_threshold_destroy(far_threshold_t* t) { delete t; }

void far_threshold_update(far_threshold_t* t, const far_pose_t* pred, const far_pose_t* reg) {
    if (!t || !pred || !reg) return;
    // deviation dT = pred^-1 * reg : rotation angle from the trace, translation in the predicted frame
    double trace = 0.0;
    for (int i = 0; i < 3; ++i)
        for (int k = 0; k < 3; ++k) trace += pred->R[3 * k + i] * reg->R[3 * k + i];
    double dt2 = 0.0;
    for (int i = 0; i < 3; ++i) {
        double c = 0.0;
        for (int k = 0; k < 3; ++k) c += pred->R[3 * k + i] * (reg->t[k] - pred->t[k]);
        dt2 += c * c;
    }
    const double cosang = std::min(1.0, std::max(-1.0, 0.5 * (trace - 1.0)));
    const double theta = std::acos(cosang);
    const double delta = std::sqrt(dt2) + 2.0 * t->max_range * std::sin(0.5 * theta);
    if (delta > t->min_motion) {
        t->sum_sq += delta * delta;
        t->count += 1;
    }
}

double far_threshold_sigma(const far_threshold_t* t) {
    if (!t) return 0.0;
    return t->count == 0 ? t->sigma0 : std::sqrt(t->sum_sq / (double)t->count);
}

}  // extern "C"
