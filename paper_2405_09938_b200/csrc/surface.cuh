// Surface state of a facet at a pulse, from what K1 left in the workspace (SURVEY.md 8(a) A1 -> A2).
//
// K1 evaluates the wave sum exactly either at every pulse of the batch (H = 1) or only at KEYFRAME
// pulses kf_j = min(j H, P-1), where it also stores the time derivatives; between keyframes the state is
// the cubic Hermite interpolant in t.  Waves are slow against the PRF (omega <= ~3 rad/s): the interpolation
// error of one component is <= A (omega h)^4 / 384 (h = keyframe spacing in seconds), and sim_create picks H
// so that the sum of these bounds stays under kKeyframeHeightTol (sim_api.cu, hard part 3).  The slopes
// only scale sigma0 (tilt modulation): they are interpolated LINEARLY, per-component error <= A_w |k_w| (omega_w h)^2 / 8
// (4 x their root-sum-square kept under kKeyframeSlopeTol by sim_create; rate rows for a cubic interpolant were tried:
// +40 % of K1 for 1e-5 of relative L2).  The oracle always evaluates exactly per pulse.
#pragma once
#include "heeps_common.cuh"

namespace heeps {

struct SurfaceArgs {
    const double *z, *zt;               // [n][F] height above centre_z and its time derivative (zt: H > 1 only)
    const float2 *slope;                // [n][F] or null (tilt modulation only)
    const float2 *slope_t;              // [n][F] or null: time derivative of the slope (cubic Hermite between keyframes; null: linear -- what K1 provides)
    const double2 *dxy, *dxy_t;         // [n][F] or null (Choppy Wave Model only)
    int32_t H;                          // 1: n = pulses of the batch; > 1: n = keyframes of the batch
    int32_t key0;                       // H > 1: index j of the first keyframe held
    int32_t n_pulses_total;             // P
};

struct SurfaceInterp {                  // per (CTA, pulse)
    size_t row0, row1;                  // rows of the two bracketing keyframes (H = 1: row0 = pulse row)
    double w00, w10, w01, w11;          // Hermite weights of z0, zt0, z1, zt1 (w10, w11 include h)
    float s;                            // (t - t0) / h
};

__device__ __forceinline__ SurfaceInterp surface_interp(const SurfaceArgs &sa, const PulseConst *pulses, int p, int pl)
{
    SurfaceInterp it;
    if (sa.H <= 1) {
        it.row0 = it.row1 = (size_t)pl;
        it.w00 = 1.0; it.w10 = it.w01 = it.w11 = 0.0; it.s = 0.f;
        return it;
    }
    const int P = sa.n_pulses_total;
    const int n_keys = (P - 1 + sa.H - 1) / sa.H + 1;
    int j = p / sa.H;
    if (j > n_keys - 2) j = n_keys - 2;
    const int k0 = min(j * sa.H, P - 1), k1 = min((j + 1) * sa.H, P - 1);
    const double t0 = pulses[k0].t, t1 = pulses[k1].t, t = pulses[p].t;
    const double h = t1 - t0;
    const double s = (h != 0.0) ? (t - t0) / h : 0.0;
    const double s2 = s * s, s3 = s2 * s;
    it.row0 = (size_t)(j - sa.key0);
    it.row1 = it.row0 + 1;
    it.w00 = 2.0 * s3 - 3.0 * s2 + 1.0;
    it.w10 = (s3 - 2.0 * s2 + s) * h;
    it.w01 = -2.0 * s3 + 3.0 * s2;
    it.w11 = (s3 - s2) * h;
    it.s = (float)s;
    return it;
}

__device__ __forceinline__ double surface_z(const SurfaceArgs &sa, const SurfaceInterp &it, size_t F, size_t f)
{
    if (sa.H <= 1) return sa.z[it.row0 * F + f];
    const size_t a = it.row0 * F + f, b = it.row1 * F + f;
    return fma(it.w00, sa.z[a], fma(it.w10, sa.zt[a], fma(it.w01, sa.z[b], it.w11 * sa.zt[b])));
}

__device__ __forceinline__ float2 surface_slope(const SurfaceArgs &sa, const SurfaceInterp &it, size_t F, size_t f)
{
    if (sa.H <= 1) return sa.slope[it.row0 * F + f];
    const size_t a = it.row0 * F + f, b = it.row1 * F + f;
    const float2 s0 = sa.slope[a], s1 = sa.slope[b];
    if (sa.slope_t) {                                   // cubic Hermite, like the height
        const float2 r0 = sa.slope_t[a], r1 = sa.slope_t[b];
        const float w00 = (float)it.w00, w10 = (float)it.w10, w01 = (float)it.w01, w11 = (float)it.w11;
        return make_float2(fmaf(w00, s0.x, fmaf(w10, r0.x, fmaf(w01, s1.x, w11 * r1.x))),
                           fmaf(w00, s0.y, fmaf(w10, r0.y, fmaf(w01, s1.y, w11 * r1.y))));
    }
    return make_float2(fmaf(it.s, s1.x - s0.x, s0.x), fmaf(it.s, s1.y - s0.y, s0.y));
}

__device__ __forceinline__ double2 surface_dxy(const SurfaceArgs &sa, const SurfaceInterp &it, size_t F, size_t f)
{
    if (sa.H <= 1) return sa.dxy[it.row0 * F + f];
    const size_t a = it.row0 * F + f, b = it.row1 * F + f;
    const double2 s0 = sa.dxy[a], d0 = sa.dxy_t[a], s1 = sa.dxy[b], d1 = sa.dxy_t[b];
    return make_double2(fma(it.w00, s0.x, fma(it.w10, d0.x, fma(it.w01, s1.x, it.w11 * d1.x))),
                        fma(it.w00, s0.y, fma(it.w10, d0.y, fma(it.w01, s1.y, it.w11 * d1.y))));
}

}  // namespace heeps
