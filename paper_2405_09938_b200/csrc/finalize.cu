// K4 -- finalize: apply the factors that were taken out of the sum,
//   exp(j 2 pi kappa (n - n_mid)^2)   facet-independent part of the chirp phase, and
//   exp(-j 2 pi f0 t0[p])            carrier phase of the reference path R0 = c0 t0[p]
// (both tabulated in fp64 at sim_create), cast to complex64 and write [c][p][n]
// (raw data output).  HBM-bound: 16 B read + 8 B written per sample.
//
// Also here: speckle-from-seed (reading G14) -- Philox4x32-10 (Salmon et al., SC'11) keyed by
// the seed, counter = facet index, Box-Muller; variance 1/2 per part.
#include "kernels.cuh"

namespace heeps {

namespace {

__global__ void __launch_bounds__(256)
finalize_kernel(DevParams prm, FinalizeArgs a, int p0, int n_pl)
{
    const int ns = prm.n_samples;
    const size_t total = (size_t)prm.n_channels * n_pl * ns;
    for (size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < total; k += (size_t)gridDim.x * blockDim.x) {
        const int n = (int)(k % ns);
        const size_t cp = k / ns;
        const int pl = (int)(cp % n_pl), c = (int)(cp / n_pl);
        const double2 v = a.acc[k];
        const double2 e = __ldg(a.chirp_n + n);
        const double2 q = __ldg(a.carrier_p + p0 + pl);
        const double fr = e.x * q.x - e.y * q.y, fi = e.x * q.y + e.y * q.x;
        float2 o;
        o.x = (float)(v.x * fr - v.y * fi);
        o.y = (float)(v.x * fi + v.y * fr);
        a.out[((size_t)c * a.n_out_pulses + a.out_pulse0 + pl) * ns + n] = o;
    }
}

__device__ __forceinline__ void philox_round(uint32_t ctr[4], const uint32_t key[2])
{
    const uint32_t hi0 = __umulhi(0xD2511F53u, ctr[0]), lo0 = 0xD2511F53u * ctr[0];
    const uint32_t hi1 = __umulhi(0xCD9E8D57u, ctr[2]), lo1 = 0xCD9E8D57u * ctr[2];
    const uint32_t n0 = hi1 ^ ctr[1] ^ key[0], n2 = hi0 ^ ctr[3] ^ key[1];
    ctr[0] = n0; ctr[1] = lo1; ctr[2] = n2; ctr[3] = lo0;
}

__global__ void __launch_bounds__(256)
speckle_kernel(float2 *xi, int64_t n, uint64_t seed)
{
    const int64_t f = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (f >= n) return;
    uint32_t ctr[4] = {(uint32_t)f, (uint32_t)((uint64_t)f >> 32), 0u, 0u};
    uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        philox_round(ctr, key);
        key[0] += 0x9E3779B9u; key[1] += 0xBB67AE85u;
    }
    // u1 in (0,1], u2 in [0,1)
    const float u1 = ((float)(ctr[0] >> 8) + 1.0f) * (1.0f / 16777216.0f);
    const float u2 = (float)(ctr[1] >> 8) * (1.0f / 16777216.0f);
    const float rad = sqrtf(-logf(u1));            // |xi|^2 ~ Exp(1): variance 1/2 per part
    float s, c;
    sincospif(2.0f * u2, &s, &c);
    xi[f] = make_float2(rad * c, rad * s);
}

__global__ void __launch_bounds__(256)
speckle_polar_kernel(const float2 *xi, uint2 *polar, int64_t n)
{
    const int64_t f = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (f >= n) return;
    const float2 v = xi[f];
    const double turns = atan2((double)v.y, (double)v.x) * 0.15915494309189535;     // [-0.5, 0.5]
    const double fr = turns - floor(turns);
    uint2 o;
    o.x = __float_as_uint(sqrtf(v.x * v.x + v.y * v.y));
    o.y = (uint32_t)(unsigned long long)(fr * 4294967296.0 + 0.5);
    polar[f] = o;
}

}  // namespace

cudaError_t launch_speckle_polar(const float2 *xi, uint2 *xi_polar, int64_t n_facets, cudaStream_t s)
{
    const int blocks = (int)((n_facets + 255) / 256);
    speckle_polar_kernel<<<blocks, 256, 0, s>>>(xi, xi_polar, n_facets);
    return cudaGetLastError();
}

cudaError_t launch_finalize(const DevParams &prm, const FinalizeArgs &a, int p0, int n_pl, cudaStream_t s)
{
    const size_t total = (size_t)prm.n_channels * n_pl * prm.n_samples;
    int blocks = (int)((total + 255) / 256);
    if (blocks > 148 * 16) blocks = 148 * 16;
    finalize_kernel<<<blocks, 256, 0, s>>>(prm, a, p0, n_pl);
    return cudaGetLastError();
}

cudaError_t launch_speckle_from_seed(float2 *xi, int64_t n_facets, uint64_t seed, cudaStream_t s)
{
    const int blocks = (int)((n_facets + 255) / 256);
    speckle_kernel<<<blocks, 256, 0, s>>>(xi, n_facets, seed);
    return cudaGetLastError();
}

}  // namespace heeps
