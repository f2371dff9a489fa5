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

}  // namespace

cudaError_t launch_finalize(const DevParams &prm, const FinalizeArgs &a, int p0, int n_pl, cudaStream_t s)
{
    const size_t total = (size_t)prm.n_channels * n_pl * prm.n_samples;
    int blocks = (int)((total + 255) / 256);
    if (blocks > 148 * 16) blocks = 148 * 16;
    finalize_kernel<<<blocks, 256, 0, s>>>(prm, a, p0, n_pl);
    return cudaGetLastError();
}

}  // namespace heeps
