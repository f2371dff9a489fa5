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

struct Leg { double r; float g; };

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
    return o;
}


}  // namespace heeps
