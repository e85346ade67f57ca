// Frame stream (include/pcamm.h, "frame stream"): consecutive projections of one treatment, each
// solve started from the coefficients predicted from the frames before it (
// DESIGN.md reading B9).  Host logic only: the solve itself is pcamm_reconstruct[_host].
#include <cmath>
#include <new>
#include <string>

#include "../../include/pcamm.h"
#include "internal.h"

struct pcamm_frames {
    pcamm_model* model = nullptr;
    int K = 0, order = 0, n = 0;                       // n: frames held, newest last
    double t[PCAMM_PREDICT_MAX_ORDER + 1] = {};
    double w[PCAMM_PREDICT_MAX_ORDER + 1][PCAMM_KMAX] = {};
    float w0[PCAMM_KMAX] = {};
};

namespace {

int bad(const char* msg) {
    pcamm::set_error(msg);
    return PCAMM_E_INVALID;
}

// Newton's divided differences through the last m of n frames (oldest first), evaluated at time tq
// (Horner from the newest node); m = 1: the last frame's w.
void extrapolate_from(int order, int K, int n, const double* t, const double (*w)[PCAMM_KMAX], const float* w0,
                      double tq, float* out) {
    if (order < 0 || n == 0) {
        for (int k = 0; k < K; ++k) out[k] = w0 ? w0[k] : 0.f;
        return;
    }
    int m = (order < n - 1 ? order : n - 1) + 1;
    for (int i = n - m; i < n && m > 1; ++i)
        for (int j = i + 1; j < n; ++j)
            if (t[i] == t[j]) m = 1;                   // equal stamps: hold
    const double* tn = t + (n - m);
    for (int k = 0; k < K; ++k) {
        double d[PCAMM_PREDICT_MAX_ORDER + 1];
        for (int i = 0; i < m; ++i) d[i] = w[n - m + i][k];
        for (int lvl = 1; lvl < m; ++lvl)              // d[i] <- f[t_{i-lvl}, ..., t_i]
            for (int i = m - 1; i >= lvl; --i) d[i] = (d[i] - d[i - 1]) / (tn[i] - tn[i - lvl]);
        double v = d[m - 1];
        for (int i = m - 2; i >= 0; --i) v = v * (tq - tn[i]) + d[i];
        out[k] = (float)v;
    }
}

void extrapolate(const pcamm_frames* s, double tq, float* out) {
    extrapolate_from(s->order, s->K, s->n, s->t, s->w, s->w0, tq, out);
}

}  // namespace

extern "C" {

int pcamm_predict_w(int32_t order, int32_t K, int32_t n, const double* t_host, const float* w_host,
                    const float* w0_host, double t, float* w_pred_host) {
    if (!w_pred_host || (n > 0 && (!t_host || !w_host))) return bad("NULL argument");
    if (K < 1 || K > PCAMM_KMAX || n < 0) return bad("K or n out of range");
    if (order < PCAMM_PREDICT_NONE || order > PCAMM_PREDICT_MAX_ORDER) return bad("predictor order outside [-1, 2]");
    if (!std::isfinite(t)) return bad("time stamp is not finite");
    constexpr int CAP = PCAMM_PREDICT_MAX_ORDER + 1;
    const int m = n < CAP ? n : CAP;                   // only the last CAP frames can matter
    double tt[CAP] = {};
    double ww[CAP][PCAMM_KMAX] = {};
    for (int i = 0; i < m; ++i) {
        tt[i] = t_host[n - m + i];
        for (int k = 0; k < K; ++k) ww[i][k] = (double)w_host[(size_t)(n - m + i) * K + k];
    }
    extrapolate_from(order, K, m, tt, ww, w0_host, t, w_pred_host);
    return PCAMM_OK;
}

int pcamm_frames_create(pcamm_model* model, int32_t order, const float* w0_host, pcamm_frames** out) {
    if (out) *out = nullptr;
    if (!model || !out) return bad("NULL argument");
    if (order < PCAMM_PREDICT_NONE || order > PCAMM_PREDICT_MAX_ORDER) return bad("predictor order outside [-1, 2]");
    pcamm_frames* s = new (std::nothrow) pcamm_frames;
    if (!s) { pcamm::set_error("out of host memory"); return PCAMM_E_NOMEM; }
    s->model = model;
    s->K = pcamm::model_K(model);
    s->order = order;
    for (int k = 0; k < s->K; ++k) {
        s->w0[k] = w0_host ? w0_host[k] : 0.f;
        if (!std::isfinite(s->w0[k])) { delete s; pcamm::set_error("w0 is not finite"); return PCAMM_E_NONFINITE; }
    }
    *out = s;
    return PCAMM_OK;
}

void pcamm_frames_destroy(pcamm_frames* s) { delete s; }

int pcamm_frames_reset(pcamm_frames* s) {
    if (!s) return bad("NULL argument");
    s->n = 0;
    return PCAMM_OK;
}

int32_t pcamm_frames_count(const pcamm_frames* s) { return s ? s->n : 0; }

int pcamm_frames_predict(const pcamm_frames* s, double t, float* w_pred_host) {
    if (!s || !w_pred_host) return bad("NULL argument");
    if (!std::isfinite(t)) return bad("time stamp is not finite");
    extrapolate(s, t, w_pred_host);
    return PCAMM_OK;
}

int pcamm_frames_push(pcamm_frames* s, const float* y, int32_t y_on_host, float angle_rad, double t,
                      const pcamm_opts* opts, float* w_out_host, float* w_init_out_host, float* volume_out_dev,
                      float* landmarks_out_host, pcamm_info* info, void* stream) {
    if (!s || !y || !w_out_host) return bad("NULL argument");
    if (!std::isfinite(t)) return bad("time stamp is not finite");
    if (s->n > 0 && t < s->t[s->n - 1]) return bad("time stamps must not decrease");
    float w_init[PCAMM_KMAX];
    extrapolate(s, t, w_init);
    for (int k = 0; k < s->K; ++k)
        if (!std::isfinite(w_init[k])) { pcamm::set_error("predicted start is not finite"); return PCAMM_E_NONFINITE; }
    float w_new[PCAMM_KMAX];
    const int rc = y_on_host ? pcamm_reconstruct_host(s->model, y, angle_rad, w_init, opts, w_new, volume_out_dev,
                                                      landmarks_out_host, info, stream)
                             : pcamm_reconstruct(s->model, y, angle_rad, w_init, opts, w_new, volume_out_dev,
                                                 landmarks_out_host, info, stream);
    if (rc < 0) return rc;
    for (int k = 0; k < s->K; ++k) w_out_host[k] = w_new[k];
    if (w_init_out_host)
        for (int k = 0; k < s->K; ++k) w_init_out_host[k] = w_init[k];
    constexpr int CAP = PCAMM_PREDICT_MAX_ORDER + 1;
    if (s->n == CAP) {
        for (int i = 1; i < CAP; ++i) {
            s->t[i - 1] = s->t[i];
            for (int k = 0; k < s->K; ++k) s->w[i - 1][k] = s->w[i][k];
        }
        s->n = CAP - 1;
    }
    s->t[s->n] = t;
    for (int k = 0; k < s->K; ++k) s->w[s->n][k] = (double)w_new[k];
    s->n += 1;
    return rc;
}

}  // extern "C"
