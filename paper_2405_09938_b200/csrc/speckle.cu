// Intra-facet speckle.
//
// Static speckle (the default; reading G13): xi_f is constant over the dwell -- an input map, or, with
// sim_scene.xi = NULL, drawn here from the seed (reading G14): Philox4x32-10 (Salmon et al., SC'11) keyed by the
// seed, counter (f, 0, 0), Box-Muller, variance 1/2 per part.
//
// Time-dependent speckle (sim_scene.speckle_tau_s > 0): eq. (7)
//     s(t) = [R(t) + i I(t)] exp(2 i pi f_s t)
// with the order-1 autoregressive model of eq. (10), stepped pulse by pulse from R(0) + i I(0) = xi_f:
//     R(t + dt) = beta R(t) + (1 - beta^2)^(1/2) R',  beta = exp(-dt / tau_s),  R' ~ N(0, variance 1/2).
// Reading G27: the innovation of facet f at pulse q is Philox4x32-10 with counter (f lo, f hi, q, 1), mapped like
// the static draw.  One thread per facet walks the pulses of a batch and writes, per pulse, the POLAR form
// {|s|, arg s in 2^-32 turns} that K2 / K2s / K2k fold into the fixed-point phase word.  The walk starts from the
// state cached after the previous batch when the batches are consecutive, else it replays from pulse 0 (the
// result depends only on (seed, f, q), never on the call pattern: sim_generate stays idempotent per pulse range).
// Bound: ALU (about 150 instructions per facet-pulse), 8 B written per facet-pulse.
#include "kernels.cuh"

namespace heeps {

namespace {

__device__ __forceinline__ void philox4x32_10(uint32_t ctr[4], uint32_t k0, uint32_t k1)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, ctr[0]), lo0 = 0xD2511F53u * ctr[0];
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, ctr[2]), lo1 = 0xCD9E8D57u * ctr[2];
        const uint32_t n0 = hi1 ^ ctr[1] ^ k0, n2 = hi0 ^ ctr[3] ^ k1;
        ctr[0] = n0; ctr[1] = lo1; ctr[2] = n2; ctr[3] = lo0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
}

// circular complex Gaussian, variance 1/2 per part, from one Philox block
__device__ __forceinline__ float2 normal_pair(uint64_t seed, uint64_t f, uint32_t c2, uint32_t c3)
{
    uint32_t ctr[4] = {(uint32_t)f, (uint32_t)(f >> 32), c2, c3};
    philox4x32_10(ctr, (uint32_t)seed, (uint32_t)(seed >> 32));
    // u1 in (0,1], u2 in [0,1)
    const float u1 = ((float)(ctr[0] >> 8) + 1.0f) * (1.0f / 16777216.0f);
    const float u2 = (float)(ctr[1] >> 8) * (1.0f / 16777216.0f);
    const float rad = sqrtf(-logf(u1));            // |xi|^2 ~ Exp(1)
    float s, c;
    sincospif(2.0f * u2, &s, &c);
    return make_float2(rad * c, rad * s);
}

__device__ __forceinline__ uint2 to_polar(float2 v, uint32_t extra_turns)
{
    const double turns = atan2((double)v.y, (double)v.x) * 0.15915494309189535;     // [-0.5, 0.5]
    const double fr = turns - floor(turns);
    uint2 o;
    o.x = __float_as_uint(sqrtf(v.x * v.x + v.y * v.y));
    o.y = (uint32_t)(unsigned long long)(fr * 4294967296.0 + 0.5) + extra_turns;
    return o;
}

// the same in fp32 for the per-pulse walk (atan2f: ~1e-7 rad, 2e-8 turns)
__device__ __forceinline__ uint2 to_polar_fast(float2 v, uint32_t extra_turns)
{
    const float turns = atan2f(v.y, v.x) * 0.15915494309189535f;                    // [-0.5, 0.5]
    uint2 o;
    o.x = __float_as_uint(sqrtf(v.x * v.x + v.y * v.y));
    o.y = (uint32_t)__float2int_rn(turns * 2147483648.0f) * 2u + extra_turns;       // 2^-32 turns, wrapping
    return o;
}

__global__ void __launch_bounds__(256)
speckle_kernel(float2 *xi, int64_t n, uint64_t seed)
{
    const int64_t f = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (f >= n) return;
    xi[f] = normal_pair(seed, (uint64_t)f, 0u, 0u);
}

__global__ void __launch_bounds__(256)
speckle_polar_kernel(const float2 *xi, uint2 *polar, int64_t n)
{
    const int64_t f = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (f >= n) return;
    polar[f] = to_polar(xi[f], 0u);
}

__global__ void __launch_bounds__(256)
speckle_ar1_kernel(SpeckleAr1Args a)
{
    const int64_t f = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (f >= a.n_facets) return;
    float2 st;
    int q;
    if (a.resume) { st = a.state[f]; q = a.p0; }            // state after pulse p0 - 1
    else { st = a.xi[f]; q = 1; }                            // replay from pulse 0
    for (; q < a.p0; ++q) {
        const float2 bg = __ldg(a.beta_g + q);
        const float2 nn = normal_pair(a.seed, (uint64_t)f, (uint32_t)q, 1u);
        st.x = fmaf(bg.x, st.x, bg.y * nn.x);
        st.y = fmaf(bg.x, st.y, bg.y * nn.y);
    }
    for (int pl = 0; pl < a.n_pl; ++pl) {
        const int p = a.p0 + pl;
        if (p > 0) {
            const float2 bg = __ldg(a.beta_g + p);
            const float2 nn = normal_pair(a.seed, (uint64_t)f, (uint32_t)p, 1u);
            st.x = fmaf(bg.x, st.x, bg.y * nn.x);
            st.y = fmaf(bg.x, st.y, bg.y * nn.y);
        }
        a.polar[(size_t)pl * a.n_facets + f] = to_polar_fast(st, __ldg(a.doppler_turns + p));
    }
    a.state[f] = st;                                         // state after pulse p0 + n_pl - 1
}

}  // namespace

cudaError_t launch_speckle_polar(const float2 *xi, uint2 *xi_polar, int64_t n_facets, cudaStream_t s)
{
    const int blocks = (int)((n_facets + 255) / 256);
    speckle_polar_kernel<<<blocks, 256, 0, s>>>(xi, xi_polar, n_facets);
    return cudaGetLastError();
}

cudaError_t launch_speckle_from_seed(float2 *xi, int64_t n_facets, uint64_t seed, cudaStream_t s)
{
    const int blocks = (int)((n_facets + 255) / 256);
    speckle_kernel<<<blocks, 256, 0, s>>>(xi, n_facets, seed);
    return cudaGetLastError();
}

cudaError_t launch_speckle_ar1(const SpeckleAr1Args &a, cudaStream_t s)
{
    if (a.n_pl <= 0) return cudaSuccess;
    const int blocks = (int)((a.n_facets + 255) / 256);
    speckle_ar1_kernel<<<blocks, 256, 0, s>>>(a);
    return cudaGetLastError();
}

}  // namespace heeps
