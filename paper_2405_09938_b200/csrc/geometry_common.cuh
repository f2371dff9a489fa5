// Device helpers shared by the two geometry kernels (geometry.cu: records for the direct path;
// moments.cu: range-slice moments for the spectral path).  SURVEY.md 8(a) A2/A3.
#pragma once
#include "heeps_common.cuh"

namespace heeps {

__device__ __forceinline__ float sinc_pi(float x)
{   // sin(pi x)/(pi x); field pattern of a uniform aperture (G5)
    if (x == 0.f) return 1.f;
    return sinpif(x) / (3.14159265358979323846f * x);
}

__device__ __forceinline__ uint32_t turns_to_u32(double x)
{   // frac(x) in 2^-32 turn units, round to nearest, wrapping
    double f = x - floor(x);
    return (uint32_t)(unsigned long long)(f * 4294967296.0 + 0.5);
}

// K3 maps the top 23 bits of the phase word to a float in [1,2) and subtracts 1.5, i.e. it sees
// (turns mod 1) - 0.5 truncated to 2^-23: bias the stored word by half a turn (centres the MUFU
// argument on [-pi, pi)) plus half an lsb of the truncation (round to nearest).
constexpr uint32_t kPhiBias = 0x80000000u + 256u;

// sqrt and reciprocal sqrt of a squared range in one go: rsqrt seed, one fused correction of the root
// (|error| <= 1 ulp of r); replaces IEEE sqrt() + 1/r (about a third of their instruction count).
__device__ __forceinline__ void root_and_inverse(double r2, double &r, double &inv)
{
    const double y = rsqrt(r2);
    const double rr = r2 * y;
    r = fma(fma(-rr, rr, r2), 0.5 * y, rr);
    inv = y;
}

__device__ __forceinline__ float sinc_pi_fast(float x)
{   // same function without sinpif/IEEE division: with n = rint(x), r = x - n in [-1/2, 1/2],
    //   sin(pi x)/(pi x) = (-1)^n [sin(pi r)/(pi r)] r / x,
    // the bracket by its Taylor series through (pi r)^10 (next term 3.6e-8 at r = 1/2).  |x| < 2^22.
    if (x == 0.f) return 1.f;
    const float n = rintf(x), r = x - n;
    const float t = r * r;
    float p = fmaf(t, -2.3460810e-3f, 2.6147848e-2f);        // -pi^10/11!, pi^8/9!
    p = fmaf(t, p, -1.9075182e-1f);                            // -pi^6/7!
    p = fmaf(t, p, 8.1174243e-1f);                             //  pi^4/5!
    p = fmaf(t, p, -1.6449341f);                               // -pi^2/3!
    p = fmaf(t, p, 1.0f);
    const float q = __fdividef(p * r, x);
    return ((int)n & 1) ? -q : q;
}

__device__ __forceinline__ uint32_t turns_to_u32_fast(double x)
{   // frac(x) in 2^-32 turn units for |x| < 2^30: the 64-bit integer conversion wraps modulo one turn
    return (uint32_t)(unsigned long long)__double2ll_rn(x * 4294967296.0);
}

struct Leg { double r; float g; double ua, ue; };    // range, analytic gain, direction cosines along azimuth / elevation

// Tabulated pattern (reading G29): bilinear interpolant of the four surrounding nodes, real and imaginary parts
// separately; zero outside the grid.  Grid coordinates in fp64 (a float direction cosine resolves only ~1e-3 of a
// fine grid's step), weights and values in fp32.
__device__ __forceinline__ float2 lut_gain(const PatternLut &L, double ua, double ue)
{
    const double gu = (ua - L.u0) * L.su, gv = (ue - L.v0) * L.sv;
    if (!(gu >= 0.0 && gu <= (double)(L.nu - 1) && gv >= 0.0 && gv <= (double)(L.nv - 1))) return make_float2(0.f, 0.f);
    const int iu = min((int)gu, L.nu - 2), iv = min((int)gv, L.nv - 2);
    const float fu = (float)(gu - iu), fv = (float)(gv - iv);
    const float2 *t = L.tab + (size_t)iv * L.nu + iu;
    const float2 t00 = __ldg(t), t01 = __ldg(t + 1), t10 = __ldg(t + L.nu), t11 = __ldg(t + L.nu + 1);
    const float w00 = (1.f - fu) * (1.f - fv), w01 = fu * (1.f - fv), w10 = (1.f - fu) * fv, w11 = fu * fv;
    return make_float2(w00 * t00.x + w01 * t01.x + w10 * t10.x + w11 * t11.x,
                       w00 * t00.y + w01 * t01.y + w10 * t10.y + w11 * t11.y);
}

// Complex gain of antenna k (0 Tx, 1 Rx): the table if there is one, else (analytic, 0).
__device__ __forceinline__ float2 gain_of(const DevParams &prm, int k, float analytic, double ua, double ue)
{
    return prm.lut[k].tab ? lut_gain(prm.lut[k], ua, ue) : make_float2(analytic, 0.f);
}

__device__ __forceinline__ float2 cmulf(float2 a, float2 b)
{
    return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x));
}

// arg z in 2^-32 turns (wrapping)
__device__ __forceinline__ uint32_t arg_u32(float2 z)
{
    return (uint32_t)__float2int_rn(atan2f(z.y, z.x) * 0.15915494309189535f * 2147483648.0f) * 2u;
}

// One antenna leg with the pieces the receive-channel series needs: d = pos - ant, r = |d|, 1/r and
// the un-normalised projections on the azimuth / elevation axes.
struct LegParts { double r, inv, da, de, dx, dy, dz; };

__device__ __forceinline__ LegParts leg_parts(const double pos[3], const double ant[3], const double ax_a[3],
                                              const double ax_e[3])
{
    LegParts o;
    o.dx = pos[0] - ant[0]; o.dy = pos[1] - ant[1]; o.dz = pos[2] - ant[2];
    root_and_inverse(fma(o.dx, o.dx, fma(o.dy, o.dy, o.dz * o.dz)), o.r, o.inv);
    o.da = fma(o.dx, ax_a[0], fma(o.dy, ax_a[1], o.dz * ax_a[2]));
    o.de = fma(o.dx, ax_e[0], fma(o.dy, ax_e[1], o.dz * ax_e[2]));
    return o;
}

__device__ __forceinline__ float pattern(double da, double de, double inv, double ap_a, double ap_e)
{   // O6: sinc(La u_a / lambda) sinc(Le u_e / lambda), direction cosines u = (d . axis) / r
    return sinc_pi_fast((float)(ap_a * (da * inv))) * sinc_pi_fast((float)(ap_e * (de * inv)));
}

// Receive phase centre c sits at rx_ref + o v^ (G8).  With d = pos - rx_ref, r = |d|:
//   r_c^2 = r^2 + X,  X = o^2 - 2 o (d . v^),  delta = X / r^2   (|delta| <= ~2|o|/r)
//   r_c   = r (1 + delta/2 - delta^2/8 + delta^3/16)            truncation 5/128 delta^4
//   1/r_c = (1/r)(1 - delta/2 + 3 delta^2/8 - 5 delta^3/16)     truncation 35/128 delta^4
// sim_create enables this only when |o| <= 1e-4 r_min (delta^4 < 3e-15: below fp64 rounding of r).
__device__ __forceinline__ void channel_leg_series(const LegParts &ref, double dv, double o, double va, double ve,
                                                   double &r_c, double &inv_c, double &da_c, double &de_c)
{
    const double X = fma(o, o, -2.0 * o * dv);
    const double dl = X * ref.inv * ref.inv;
    r_c = fma(ref.r, dl * fma(dl, fma(dl, 0.0625, -0.125), 0.5), ref.r);
    inv_c = fma(ref.inv, dl * fma(dl, fma(dl, -0.3125, 0.375), -0.5), ref.inv);
    da_c = fma(-o, va, ref.da);
    de_c = fma(-o, ve, ref.de);
}

__device__ __forceinline__ Leg leg(const double pos[3], const double ant[3], const double ax_a[3],
                                   const double ax_e[3], double ap_a, double ap_e)
{
    double dx = pos[0] - ant[0], dy = pos[1] - ant[1], dz = pos[2] - ant[2];
    double r = sqrt(dx * dx + dy * dy + dz * dz);
    double inv = 1.0 / r;
    double ua = (dx * ax_a[0] + dy * ax_a[1] + dz * ax_a[2]) * inv;    // direction cosines (O6)
    double ue = (dx * ax_e[0] + dy * ax_e[1] + dz * ax_e[2]) * inv;
    Leg o;
    o.r = r;
    o.g = sinc_pi((float)(ap_a * ua)) * sinc_pi((float)(ap_e * ue));
    o.ua = ua; o.ue = ue;
    return o;
}


}  // namespace heeps
