// kf_kernels.cuh -- the float32 helix Kalman filter of K5 (prior, transport, gate, update) and small K6 helpers.
// Every float expression is parenthesised exactly as DESIGN.md "O5" writes it and compiled with -fmad=false:
// the gates, windows and arg-mins then take the same decisions as the strict-float32 reference.
#pragma once
#include "common.cuh"

namespace tpc {

// Fit state: y, z, sin phi, tg lambda (dz/dS), q/pT and the lower triangle of the covariance.
struct Fit {
    float y, z, s, t, q;
    float c00, c10, c11, c20, c21, c22, c30, c31, c32, c33, c40, c41, c42, c43, c44;
    float chi2;
    int n;
};

__device__ __forceinline__ void fit_prior(Fit& f, const Const& c) {
    f.c00 = c.sigma_y2; f.c11 = c.sigma_z2; f.c22 = c.p.var_s; f.c33 = c.p.var_t; f.c44 = c.p.var_q;
    f.c10 = f.c20 = f.c21 = f.c30 = f.c31 = f.c32 = f.c40 = f.c41 = f.c42 = f.c43 = 0.f;
    f.chi2 = 0.f;
}

// Helix transport x -> x1.  false (fit untouched) if |sin phi| leaves [-s_max, s_max].
__device__ __forceinline__ bool fit_transport(Fit& f, float x, float x1, const Const& c) {
    const float kB = c.kB;
    const float dx = x1 - x;
    const float kap = kB * f.q;
    const float s = f.s, s1 = s + kap * dx;
    if (fabsf(s) > c.p.sin_max) return false;
    if (fabsf(s1) > c.p.sin_max) return false;
    const float c0 = sqrtf(1.f - s * s), c1 = sqrtf(1.f - s1 * s1);
    const float icc = 1.f / (c0 + c1), ic0 = 1.f / c0, ic1 = 1.f / c1;
    const float dy = dx * ((s + s1) * icc);
    const float dl2 = dx * dx + dy * dy;
    const float adl = sqrtf(dl2);
    const float dl = (dx < 0.f) ? -adl : adl;
    const float idl = 1.f / dl;
    const float u = kap * dl, u2 = u * u;
    const float c24 = 1.f / 24.f, c640 = 3.f / 640.f, c12 = 1.f / 12.f;
    const float dS = dl * (1.f + u2 * (c24 + u2 * c640));
    const float ccd = 1.f + (c0 * c1 + s * s1);
    // Jacobian rows y: (1 0 a 0 b), z: (0 1 cc d e), s: (0 0 1 0 ff)
    const float a = dx * ccd * icc * ic0 * ic1;
    const float b = kB * (dx * dx) * ccd * ic1 * icc * icc;
    const float cc = f.t * dy * ic0 * ic1;
    const float d = dS;
    const float e = f.t * ((dy * idl) * b + (kB * kap) * (dl * dl2) * c12);
    const float ff = kB * dx;
    f.y = f.y + dy; f.z = f.z + f.t * dS; f.s = s1;
    // M = F C, terms added in ascending column index of F
    const float m00 = f.c00 + a * f.c20 + b * f.c40;
    const float m02 = f.c20 + a * f.c22 + b * f.c42;
    const float m04 = f.c40 + a * f.c42 + b * f.c44;
    const float m10 = f.c10 + cc * f.c20 + d * f.c30 + e * f.c40;
    const float m11 = f.c11 + cc * f.c21 + d * f.c31 + e * f.c41;
    const float m12 = f.c21 + cc * f.c22 + d * f.c32 + e * f.c42;
    const float m13 = f.c31 + cc * f.c32 + d * f.c33 + e * f.c43;
    const float m14 = f.c41 + cc * f.c42 + d * f.c43 + e * f.c44;
    const float m20 = f.c20 + ff * f.c40, m21 = f.c21 + ff * f.c41, m22 = f.c22 + ff * f.c42;
    const float m23 = f.c32 + ff * f.c43, m24 = f.c42 + ff * f.c44;
    const float m30 = f.c30, m31 = f.c31, m32 = f.c32, m33 = f.c33, m34 = f.c43;
    const float m40 = f.c40, m41 = f.c41, m42 = f.c42, m43 = f.c43, m44 = f.c44;
    // C' = M F^T, lower triangle, terms added in ascending column index
    f.c00 = m00 + m02 * a + m04 * b;
    f.c10 = m10 + m12 * a + m14 * b;
    f.c11 = m11 + m12 * cc + m13 * d + m14 * e;
    f.c20 = m20 + m22 * a + m24 * b;
    f.c21 = m21 + m22 * cc + m23 * d + m24 * e;
    f.c22 = m22 + m24 * ff;
    f.c30 = m30 + m32 * a + m34 * b;
    f.c31 = m31 + m32 * cc + m33 * d + m34 * e;
    f.c32 = m32 + m34 * ff;
    f.c33 = m33;
    f.c40 = m40 + m42 * a + m44 * b;
    f.c41 = m41 + m42 * cc + m43 * d + m44 * e;
    f.c42 = m42 + m44 * ff;
    f.c43 = m43;
    f.c44 = m44;
    return true;
}

// gate value of a measurement against the predicted state
__device__ __forceinline__ float fit_gate(const Fit& f, float my, float mz, const Const& c) {
    const float ry = my - f.y, rz = mz - f.z;
    const float wy = 1.f / (f.c00 + c.sigma_y2);
    const float wz = 1.f / (f.c11 + c.sigma_z2);
    return (ry * ry) * wy + (rz * rz) * wz;
}

// two scalar updates, y then z; iwy = 1 / (C_yy + sigma_y^2) of the predicted state
__device__ __forceinline__ void fit_update(Fit& f, float my, float mz, float iwy, const Const& c) {
    {
        const float r = my - f.y;
        const float w = iwy;
        const float k0 = f.c00, k1 = f.c10, k2 = f.c20, k3 = f.c30, k4 = f.c40;
        const float g0 = k0 * w, g1 = k1 * w, g2 = k2 * w, g3 = k3 * w, g4 = k4 * w;
        f.y = f.y + g0 * r; f.z = f.z + g1 * r; f.s = f.s + g2 * r; f.t = f.t + g3 * r; f.q = f.q + g4 * r;
        f.c00 = f.c00 - g0 * k0;
        f.c10 = f.c10 - g1 * k0; f.c11 = f.c11 - g1 * k1;
        f.c20 = f.c20 - g2 * k0; f.c21 = f.c21 - g2 * k1; f.c22 = f.c22 - g2 * k2;
        f.c30 = f.c30 - g3 * k0; f.c31 = f.c31 - g3 * k1; f.c32 = f.c32 - g3 * k2; f.c33 = f.c33 - g3 * k3;
        f.c40 = f.c40 - g4 * k0; f.c41 = f.c41 - g4 * k1; f.c42 = f.c42 - g4 * k2; f.c43 = f.c43 - g4 * k3;
        f.c44 = f.c44 - g4 * k4;
        f.chi2 = f.chi2 + (r * r) * w;
    }
    {
        const float r = mz - f.z;
        const float w = 1.f / (f.c11 + c.sigma_z2);
        const float k0 = f.c10, k1 = f.c11, k2 = f.c21, k3 = f.c31, k4 = f.c41;
        const float g0 = k0 * w, g1 = k1 * w, g2 = k2 * w, g3 = k3 * w, g4 = k4 * w;
        f.y = f.y + g0 * r; f.z = f.z + g1 * r; f.s = f.s + g2 * r; f.t = f.t + g3 * r; f.q = f.q + g4 * r;
        f.c00 = f.c00 - g0 * k0;
        f.c10 = f.c10 - g1 * k0; f.c11 = f.c11 - g1 * k1;
        f.c20 = f.c20 - g2 * k0; f.c21 = f.c21 - g2 * k1; f.c22 = f.c22 - g2 * k2;
        f.c30 = f.c30 - g3 * k0; f.c31 = f.c31 - g3 * k1; f.c32 = f.c32 - g3 * k2; f.c33 = f.c33 - g3 * k3;
        f.c40 = f.c40 - g4 * k0; f.c41 = f.c41 - g4 * k1; f.c42 = f.c42 - g4 * k2; f.c43 = f.c43 - g4 * k3;
        f.c44 = f.c44 - g4 * k4;
        f.chi2 = f.chi2 + (r * r) * w;
    }
    f.n++;
}

// selection key of tracklet i: more hits first, then the lower canonical id within the sector task
__device__ __forceinline__ uint32_t tl_key(const View& v, int i, int nh, int task_bin0) {
    const int id_in_task = i - v.seed_start[task_bin0];
    return ((uint32_t)nh << 24) | (uint32_t)(0xffffff - id_in_task);
}

// track / hit offsets of every event (tracks of one event are contiguous: seeds are ordered by task)
__global__ void k_event_offsets(const View v, int bins_per_event) {
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e > v.n_events) return;
    const int S = min(v.seed_start[v.n_bins], v.S_cap);
    const int s = min(v.seed_start[e * bins_per_event], S);
    v.ev_off[e] = v.trk_scan[s];
    v.ev_off[v.n_events + 1 + e] = v.hit_scan[s];
    if (e == v.n_events) { v.cnt[CNT_TRACKS] = (unsigned long long)v.trk_scan[s]; v.cnt[CNT_TRACK_HITS] = (unsigned long long)v.hit_scan[s]; }
}

}  // namespace tpc
