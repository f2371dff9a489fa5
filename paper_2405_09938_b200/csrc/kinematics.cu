// K1 -- facet kinematics (the resolved surface is a sum of
// wave components, linear by default, Choppy-Wave horizontal displacement by flag).
//
// On the regular facet grid the phase  psi = kx x_i + ky y_j - omega t_p + phase  is separable,
// so  A cos(psi) + j A sin(psi) = X[w][i] * Y[w][j] * T[w][p]  with three small fp64 phasor tables
// built once at sim_create.  Per facet-component this is one complex multiply-add in fp64
// instead of a sincos; fp64 because the height feeds the carrier phase (1 mrad = 8.8 um of path,
// SURVEY.md §7 hard part 2).  Slopes only scale sigma0 and stay fp32.
//
// Layout: block = 64 (i) x 4 (j) facets of one pulse; the 4 x Nw products Y*T are formed once per
// block in shared memory and broadcast; X[w][i] is read coalesced (i fastest) and stays L1/L2
// resident (Nw*nx*16 B <= 16 MB).
// Bound: FP64 pipe, 4 DFMA per facet-component (+2 FFMA with slopes).
//
// Keyframes (surface.cuh): with H > 1 the kernel runs only at the keyframe pulses min(j H, P-1) and also
// writes the time derivatives (d/dt of A cos(psi) is A omega sin(psi)), from which K2 interpolates.
#include "kernels.cuh"

namespace heeps {

namespace {

constexpr int kBX = 64, kBY = 4;

template <bool kSlope, bool kChoppy, bool kRate>
__global__ void __launch_bounds__(kBX * kBY)
kinematics_kernel(DevParams prm, KinematicsArgs a, int first)
{
    extern __shared__ double2 smem_yt[];               // [kBY][Nw] then wk [Nw] as float4
    const int nw = prm.n_waves;
    float4 *s_wk = reinterpret_cast<float4 *>(smem_yt + kBY * nw);
    // row `pl` of the outputs holds pulse p: the batch's pulses (H = 1) or its keyframes (H > 1)
    const int pl = blockIdx.z;
    const int p = kRate ? min((first + pl) * a.H, a.n_pulses_total - 1) : first + pl;
    const int j0 = blockIdx.y * kBY;
    const int tid = threadIdx.y * kBX + threadIdx.x;

    for (int idx = tid; idx < kBY * nw; idx += kBX * kBY) {
        int r = idx / nw, w = idx - r * nw;
        int j = min(j0 + r, prm.ny - 1);
        double2 y = a.yt[(size_t)w * prm.ny + j];
        double2 t = a.tt[(size_t)w * a.n_pulses_total + p];
        smem_yt[idx] = make_double2(y.x * t.x - y.y * t.y, y.x * t.y + y.y * t.x);
    }
    if (kSlope || kChoppy || kRate)
        for (int w = tid; w < nw; w += kBX * kBY) s_wk[w] = a.wk[w];
    __syncthreads();

    const int i = blockIdx.x * kBX + threadIdx.x;
    const int j = j0 + threadIdx.y;
    if (i >= prm.nx || j >= prm.ny) return;
    const double2 *yt = smem_yt + threadIdx.y * nw;
    const double2 *xt = a.xt + i;

    double z = 0.0, dx = 0.0, dy = 0.0, zt = 0.0, dxt = 0.0, dyt = 0.0;
    float sx = 0.f, sy = 0.f, sxt = 0.f, syt = 0.f;
#pragma unroll 4
    for (int w = 0; w < nw; ++w) {
        double2 x = __ldg(xt + (size_t)w * prm.nx);
        double2 y = yt[w];
        const double re = fma(x.x, y.x, -x.y * y.y);          // A cos(psi)
        z += re;
        if (kSlope || kChoppy || kRate) {
            double im = fma(x.x, y.y, x.y * y.x);             // A sin(psi)
            float4 k = s_wk[w];
            const double om = kRate ? a.omega[w] : 0.0;
            if (kRate) zt = fma(om, im, zt);                  // d/dt A cos(psi) = A omega sin(psi)
            if (kSlope) {
                float imf = (float)im;
                sx = fmaf(-k.x, imf, sx);                     // grad z = -sum A k sin(psi)
                sy = fmaf(-k.y, imf, sy);
                if (kRate) {
                    const float wre = (float)(om * re);
                    sxt = fmaf(k.x, wre, sxt);
                    syt = fmaf(k.y, wre, syt);
                }
            }
            if (kChoppy) {
                dx = fma(-(double)k.z, im, dx);               // D_h = -sum A k^ sin(psi)
                dy = fma(-(double)k.w, im, dy);
                if (kRate) {
                    dxt = fma((double)k.z * om, re, dxt);
                    dyt = fma((double)k.w * om, re, dyt);
                }
            }
        }
    }
    const size_t f = (size_t)pl * prm.nx * prm.ny + (size_t)j * prm.nx + i;
    a.z[f] = z;
    if (kSlope) a.slope[f] = make_float2(sx, sy);
    if (kChoppy) a.dxy[f] = make_double2(dx, dy);
    if (kRate) {
        a.zt[f] = zt;
        if (kSlope) a.slope_t[f] = make_float2(sxt, syt);
        if (kChoppy) a.dxy_t[f] = make_double2(dxt, dyt);
    }
}

// Slope of every facet at pulse p as K2 sees it (interpolated between keyframes); sim_debug_facets only.
__global__ void __launch_bounds__(256)
surface_slope_kernel(DevParams prm, SurfaceArgs sa, const PulseConst *pulses, int p, float2 *out)
{
    const size_t F = (size_t)prm.nx * prm.ny;
    const size_t f = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (f >= F) return;
    const SurfaceInterp it = surface_interp(sa, pulses, p, 0);
    out[f] = surface_slope(sa, it, F, f);
}

}  // namespace

cudaError_t launch_surface_slope(const DevParams &prm, const SurfaceArgs &sa, const PulseConst *pulses, int p,
                                 float2 *out, cudaStream_t s)
{
    const size_t F = (size_t)prm.nx * prm.ny;
    surface_slope_kernel<<<(unsigned)((F + 255) / 256), 256, 0, s>>>(prm, sa, pulses, p, out);
    return cudaGetLastError();
}

cudaError_t launch_kinematics(const DevParams &prm, const KinematicsArgs &a, int first, int n_rows, cudaStream_t s)
{
    if (n_rows <= 0) return cudaSuccess;
    const int n_pl = n_rows;
    dim3 block(kBX, kBY);
    dim3 grid((prm.nx + kBX - 1) / kBX, (prm.ny + kBY - 1) / kBY, n_pl);
    size_t smem = (size_t)kBY * prm.n_waves * sizeof(double2) + (size_t)prm.n_waves * sizeof(float4);
    const bool slope = a.slope != nullptr, choppy = a.dxy != nullptr;
    auto launch = [&](auto kern) {
        if (smem > 48 * 1024)
            cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        kern<<<grid, block, smem, s>>>(prm, a, first);
    };
    const bool rate = a.H > 1;
    if (rate) {
        if (slope && choppy) launch(kinematics_kernel<true, true, true>);
        else if (slope)      launch(kinematics_kernel<true, false, true>);
        else if (choppy)     launch(kinematics_kernel<false, true, true>);
        else                 launch(kinematics_kernel<false, false, true>);
    } else {
        if (slope && choppy) launch(kinematics_kernel<true, true, false>);
        else if (slope)      launch(kinematics_kernel<true, false, false>);
        else if (choppy)     launch(kinematics_kernel<false, true, false>);
        else                 launch(kinematics_kernel<false, false, false>);
    }
    return cudaGetLastError();
}

}  // namespace heeps
