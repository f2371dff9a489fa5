// K1 -- facet kinematics (the resolved surface is a sum of
// wave components, linear by default, Choppy-Wave horizontal displacement by flag).
//
// On the regular facet grid the phase  psi = kx x_i + ky y_j - omega t_p + phase  is separable,
// so  A cos(psi) + j A sin(psi) = X[w][i] * Y[w][j] * T[w][p]  with three small fp64 phasor tables
// built once at sim_create.  Per facet-component this is one complex multiply-add in fp64
// instead of a sincos; fp64 because the height feeds the carrier phase (1 mrad = 8.8 um of path,
// SURVEY.md §7 hard part 2).  Slopes only scale sigma0 and stay fp32.
//
// Layout: block = 64 (i) x 8 (j) facets x up to kPK consecutive rows (pulses or keyframes).  A thread owns two facets
// of the same column i (they share X[w][i] and every shared-memory table load); per facet:
// per wave component it forms c = X[w][i] * Y[w][j] once (X read coalesced from L2, Y from shared memory) and
// then runs over the kPK rows, multiplying by T[w][p] from shared memory (broadcast).  Only the HEIGHT (and the
// CWM displacement) is accumulated in fp64 -- 2 DFMA per facet-component-row; the time derivative and the slopes
// (linear between keyframes: no slope rates) are fp32 products of (float)c with a float copy of T (the rate enters the Hermite interpolant
// scaled by h/8 ~ 1e-3 s, the slopes only scale sigma0).  Wave components are processed in chunks of kWCh so
// that the tables fit 48 KB of shared memory for any Nw.
// Bound: 2 DFMA per facet-component-row (6 with CWM) next to 4 FP32 instructions with slopes and rates; measured
// (profiles/r1_v10): FP64 pipe 20 %, shared-memory data path 68 % -- the broadcast T-table loads (one LDS.128 +
// one LDS.64 per component-row and warp) are what binds; next step: two facets per thread or fp64 MMA fragments.
//
// Keyframes (surface.cuh): with H > 1 the kernel runs only at the keyframe pulses min(j H, P-1) and also
// writes the time derivatives (d/dt of A cos(psi) is A omega sin(psi)), from which K2 interpolates.
// Decoupled keyframes (sim_api.cu choose_coarse_spacing): for the keyframed geometry kernel the wave sums are evaluated at
// a multiple of its spacing, with second time derivatives (kRate2), and surface_refine_kernel (K1b) below writes the
// rows at its spacing from them by quintic / cubic Hermite interpolation.
#include <algorithm>
#include <type_traits>

#include "kernels.cuh"

namespace heeps {

namespace {

constexpr int kBX = 64, kBY = 4;
constexpr int kPK = 6;        // most rows per thread (the kernel is instantiated for 4..6; 2 x 6 rows of accumulators = 128 registers)
constexpr int kWCh = 128;     // wave components per shared-memory chunk
constexpr int kNF = 2;        // facets per thread (same i, rows kBY apart): they share X[w][i] and the T-table loads

// square of the weight of eq. (2), in the paper's expanded form: w_x = |x^i - x|/L, w_y = |y^i - y|/L
__device__ __forceinline__ double weight2(double wx, double wy) { return __dadd_rn(__dadd_rn(1.0 - wx, -wy), __dmul_rn(wx, wy)); }

// kRate2 (with kRate): also the SECOND time derivative of the height and the rate of the slopes -- the keyframe rows of
// the decoupled scheme (sim_api.cu: K1 at R x the spacing of the geometry kernel; quintic Hermite for the height, cubic
// Hermite for the slopes between them).
template <int NK, bool kSlope, bool kChoppy, bool kRate, bool kHetero, bool kRate2 = false>
__global__ void __launch_bounds__(kBX * kBY)
kinematics_kernel(DevParams prm, KinematicsArgs a, int first, int n_rows)
{
    __shared__ double2 s_y[kBY * kNF][kWCh];
    __shared__ double2 s_t[kWCh][NK];
    __shared__ float2 s_tf[kWCh][NK];
    __shared__ float4 s_wk[kWCh];
    __shared__ float s_om[kWCh];

    const int nw = prm.n_waves;
    const int row0 = blockIdx.z * NK;                  // first output row of this block
    const int nk = min(NK, n_rows - row0);             // rows this block stores (the last block recomputes its last row)
    const int tid = threadIdx.y * kBX + threadIdx.x;
    // Heterogeneous surface: a block stays inside one cell TL of the node lattice, so that its four
    // corner tiles T2L are the same for all its facets.  Homogeneous surface: one cell, one "corner" of weight 1.
    constexpr bool hetero = kHetero;
    int cell_a = 0, cell_b = 0, i_lo = 0, i_hi = prm.nx, j_lo = 0, j_hi = prm.ny;
    // blockIdx.x runs over the ROW blocks (j), blockIdx.y over the column blocks (i): blocks that are scheduled together
    // share their 64 X columns (262 KB for 256 components) and stream the Y rows, 8x less L2 traffic than the other
    // way round for a 64 x 8 block (the tables are tens of megabytes on the large grids)
    const int gbx = blockIdx.y, gby = blockIdx.x;
    int bx = gbx, by = gby;
    if (hetero) {
        cell_a = gbx / a.chunks_x; bx = gbx - cell_a * a.chunks_x;
        cell_b = gby / a.chunks_y; by = gby - cell_b * a.chunks_y;
        // facet i belongs to cell floor((i d) / L), in exactly this arithmetic (the weights of eq. (2) have an infinite
        // slope at the far edge of a cell: a facet that rounding puts on the other side of a node line would see a
        // weight of 1e-8 instead of 0).  first(a) = the smallest index whose cell is >= a.
        const double d = prm.spacing, L = a.node_spacing;
        auto first = [&](int cell, int n) {
            int k = min(n, max(0, (int)ceil(cell * (L / d))));
            while (k > 0 && floor(((k - 1) * d) / L) >= (double)cell) --k;
            while (k < n && floor((k * d) / L) < (double)cell) ++k;
            return k;
        };
        i_lo = first(cell_a, prm.nx); j_lo = first(cell_b, prm.ny);
        if (cell_a < a.nodes_x - 2) i_hi = first(cell_a + 1, prm.nx);
        if (cell_b < a.nodes_y - 2) j_hi = first(cell_b + 1, prm.ny);
    }
    const int j0 = j_lo + by * (kBY * kNF);
    const int i = i_lo + bx * kBX + threadIdx.x;
    if (i_lo + bx * kBX >= i_hi || j0 >= j_hi) return;     // block-uniform: this chunk of the cell holds no facet
    // facet u of the thread: (i, j0 + threadIdx.y + u kBY); both share X[w][i] and every T-table load
    bool valid[kNF];
#pragma unroll
    for (int u = 0; u < kNF; ++u) valid[u] = i < i_hi && j0 + threadIdx.y + u * kBY < j_hi;
    // position inside the cell, in lattice steps (weights of eq. (2))
    double fx = 0.0, fy[kNF];
#pragma unroll
    for (int u = 0; u < kNF; ++u) fy[u] = 0.0;
    if (hetero) {
        fx = fmin(fmax((i * prm.spacing) / a.node_spacing - cell_a, 0.0), 1.0);
#pragma unroll
        for (int u = 0; u < kNF; ++u)
            fy[u] = fmin(fmax(((j0 + threadIdx.y + u * kBY) * prm.spacing) / a.node_spacing - cell_b, 0.0), 1.0);
    }

    double z[kNF][NK], dx[kNF][NK], dy[kNF][NK];
    float zt[kNF][NK], dxt[kNF][NK], dyt[kNF][NK];
    float2 sxy[kNF][NK];
    constexpr int NK2 = kRate2 ? NK : 1;
    float ztt[kNF][NK2];
    float2 sxyt[kNF][NK2];
#pragma unroll
    for (int u = 0; u < kNF; ++u)
#pragma unroll
        for (int k = 0; k < NK; ++k) {
            z[u][k] = dx[u][k] = dy[u][k] = 0.0;
            zt[u][k] = dxt[u][k] = dyt[u][k] = 0.f; sxy[u][k] = make_float2(0.f, 0.f);
            if (kRate2) { ztt[u][k] = 0.f; sxyt[u][k] = make_float2(0.f, 0.f); }
        }

    for (int corner = 0; corner < (hetero ? 4 : 1); ++corner) {
    // tables of this corner's node (the homogeneous tile T2L_i) and the facets' weights W^i of eq. (2)
    const int ca = corner & 1, cb = corner >> 1;
    const size_t node = hetero ? (size_t)(cell_b + cb) * a.nodes_x + (cell_a + ca) : 0;
    const double2 *n_xt = a.xt + node * nw * prm.nx, *n_yt = a.yt + node * nw * prm.ny;
    const double2 *n_tt = a.tt + node * nw * a.n_pulses_total;
    const float4 *n_wk = a.wk + node * nw;
    const double *n_om = a.omega + node * nw;
    double wgt[kNF];
#pragma unroll
    for (int u = 0; u < kNF; ++u)
        wgt[u] = hetero ? sqrt(fmax(0.0, weight2(ca ? 1.0 - fx : fx, cb ? 1.0 - fy[u] : fy[u]))) : 1.0;
    for (int w0 = 0; w0 < nw; w0 += kWCh) {
        const int nwc = min(kWCh, nw - w0);
        __syncthreads();                               // the previous chunk's tables are no longer read
        for (int idx = tid; idx < kBY * kNF * nwc; idx += kBX * kBY) {
            const int r = idx / nwc, w = idx - r * nwc;
            s_y[r][w] = n_yt[(size_t)(w0 + w) * prm.ny + min(j0 + r, prm.ny - 1)];
        }
        for (int idx = tid; idx < nwc * NK; idx += kBX * kBY) {
            const int w = idx / NK, k = idx - w * NK;
            const int row = min(row0 + min(k, nk - 1), n_rows - 1);
            // row `row` of the outputs holds pulse p: the batch's pulses (H = 1) or its keyframes (H > 1)
            const int p = kRate ? min((first + row) * a.H, a.n_pulses_total - 1) : first + row;
            const double2 t = n_tt[(size_t)(w0 + w) * a.n_pulses_total + p];
            s_t[w][k] = t;
            s_tf[w][k] = make_float2((float)t.x, (float)t.y);
        }
        if (kSlope || kChoppy || kRate)
            for (int w = tid; w < nwc; w += kBX * kBY) {
                s_wk[w] = n_wk[w0 + w];
                s_om[w] = kRate ? (float)n_om[w0 + w] : 0.f;
            }
        __syncthreads();
        if (!valid[0]) continue;                       // valid[1] implies valid[0]; no barrier is skipped: `continue` is after both
        const double2 *xt = n_xt + (size_t)w0 * prm.nx + i;
#pragma unroll 2
        for (int w = 0; w < nwc; ++w) {
            const double2 x = __ldg(xt + (size_t)w * prm.nx);
            double cr[kNF], ci[kNF];
            float cfr[kNF], cfi[kNF];
#pragma unroll
            for (int u = 0; u < kNF; ++u) {
                const double2 y = s_y[threadIdx.y + u * kBY][w];
                cr[u] = wgt[u] * fma(x.x, y.x, -x.y * y.y);                            // W A exp(j (kx x + ky y + phase))
                ci[u] = wgt[u] * fma(x.x, y.y, x.y * y.x);
                cfr[u] = (float)cr[u]; cfi[u] = (float)ci[u];
            }
            float om = 0.f;
            float4 k4 = make_float4(0.f, 0.f, 0.f, 0.f);
            if (kSlope || kChoppy || kRate) { k4 = s_wk[w]; om = s_om[w]; }
            const float2 nk2 = make_float2(-k4.x, -k4.y);
#pragma unroll
            for (int k = 0; k < NK; ++k) {
                const double2 t = s_t[w][k];
                float2 tf = make_float2(0.f, 0.f);
                if (kSlope || kRate) tf = s_tf[w][k];
#pragma unroll
                for (int u = 0; u < kNF; ++u) {
                    z[u][k] = fma(cr[u], t.x, z[u][k]);                   // A cos(psi)
                    z[u][k] = fma(-ci[u], t.y, z[u][k]);
                    if (kChoppy) {
                        const double im = fma(cr[u], t.y, ci[u] * t.x);  // A sin(psi)
                        dx[u][k] = fma(-(double)k4.z, im, dx[u][k]);     // D_h = -sum A k^ sin(psi)
                        dy[u][k] = fma(-(double)k4.w, im, dy[u][k]);
                    }
                    if (kSlope || kRate) {
                        const float imf = fmaf(cfr[u], tf.y, cfi[u] * tf.x);
                        if (kRate) zt[u][k] = fmaf(om, imf, zt[u][k]);    // d/dt A cos(psi) = A omega sin(psi)
                        if (kSlope) sxy[u][k] = __ffma2_rn(nk2, make_float2(imf, imf), sxy[u][k]);   // grad z = -sum A k sin(psi)
                        if ((kChoppy || kRate2) && kRate) {
                            const float wre = om * fmaf(cfr[u], tf.x, -cfi[u] * tf.y);   // omega A cos(psi)
                            if (kChoppy) { dxt[u][k] = fmaf(k4.z, wre, dxt[u][k]); dyt[u][k] = fmaf(k4.w, wre, dyt[u][k]); }
                            if (kRate2) {
                                ztt[u][kRate2 ? k : 0] = fmaf(-om, wre, ztt[u][kRate2 ? k : 0]);      // d2/dt2 A cos(psi) = -A omega^2 cos(psi)
                                // d/dt grad z = d/dt (-A k sin(psi)) = A k omega cos(psi)   (psi = ... - omega t)
                                if (kSlope) sxyt[u][kRate2 ? k : 0] = __ffma2_rn(make_float2(k4.x, k4.y), make_float2(wre, wre), sxyt[u][kRate2 ? k : 0]);
                            }
                        }
                    }
                }
            }
        }
    }
    }
    const size_t F = (size_t)prm.nx * prm.ny;
#pragma unroll
    for (int u = 0; u < kNF; ++u) {
        if (!valid[u]) continue;
        const int j = j0 + threadIdx.y + u * kBY;
#pragma unroll
        for (int k = 0; k < NK; ++k) {
            if (k >= nk) break;
            const size_t f = (size_t)(row0 + k) * F + (size_t)j * prm.nx + i;
            a.z[f] = z[u][k];
            if (kSlope) a.slope[f] = sxy[u][k];
            if (kChoppy) a.dxy[f] = make_double2(dx[u][k], dy[u][k]);
            if (kRate2) {
                a.ztt[f] = ztt[u][kRate2 ? k : 0];
                if (kSlope) a.slope_t[f] = sxyt[u][kRate2 ? k : 0];
            }
            if (kRate) {
                a.zt[f] = (double)zt[u][k];
                if (kChoppy) a.dxy_t[f] = make_double2((double)dxt[u][k], (double)dyt[u][k]);
            }
        }
    }
}

// K1b -- keyframe rows at spacing H from K1's coarse rows at spacing H1 = R H (decoupled keyframes, sim_api.cu
// choose_coarse_spacing): height and its rate by the QUINTIC Hermite interpolant of (z, dz/dt, d2z/dt2) at the two coarse
// keyframes around, slopes by the cubic Hermite of (slope, its rate).  One thread per facet walks the output rows and
// keeps the two coarse rows in registers; HBM-bound: 36 B read per facet and coarse row, 24 B written per output row.
__global__ void __launch_bounds__(256)
surface_refine_kernel(SurfaceRefineArgs a)
{
    const size_t F = a.n_facets;
    const size_t f = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (f >= F) return;
    const int P = a.n_pulses_total, H = a.H, H1 = a.H1;
    const int n_keys1 = (P - 1 + H1 - 1) / H1 + 1;
    int m_cur = -1;
    double z0 = 0, v0 = 0, a0 = 0, z1 = 0, v1 = 0, a1 = 0, t0 = 0, hh = 1;
    float2 s0 = make_float2(0.f, 0.f), r0 = s0, s1 = s0, r1 = s0;
    for (int r = 0; r < a.n_rows; ++r) {
        const int k = min((a.first + r) * H, P - 1);                       // pulse of output row r
        const int m = min(k / H1, n_keys1 - 2);
        if (m != m_cur) {
            const size_t c0 = (size_t)(m - a.first1) * F + f, c1 = c0 + F;
            if (m == m_cur + 1 && m_cur >= 0) { z0 = z1; v0 = v1; a0 = a1; s0 = s1; r0 = r1; }
            else { z0 = a.zc[c0]; v0 = a.ztc[c0]; a0 = (double)a.zttc[c0]; if (a.slopec) { s0 = a.slopec[c0]; r0 = a.slope_tc[c0]; } }
            z1 = a.zc[c1]; v1 = a.ztc[c1]; a1 = (double)a.zttc[c1];
            if (a.slopec) { s1 = a.slopec[c1]; r1 = a.slope_tc[c1]; }
            const int q0 = min(m * H1, P - 1), q1 = min((m + 1) * H1, P - 1);
            t0 = a.pulses[q0].t; hh = a.pulses[q1].t - t0;
            m_cur = m;
        }
        const double x = (a.pulses[k].t - t0) / hh, x2 = x * x, x3 = x2 * x, x4 = x3 * x, x5 = x4 * x;
        const double w0 = 1.0 - 10.0 * x3 + 15.0 * x4 - 6.0 * x5, w5 = 10.0 * x3 - 15.0 * x4 + 6.0 * x5;
        const double w1 = (x - 6.0 * x3 + 8.0 * x4 - 3.0 * x5) * hh, w4 = (-4.0 * x3 + 7.0 * x4 - 3.0 * x5) * hh;
        const double w2 = 0.5 * (x2 - 3.0 * x3 + 3.0 * x4 - x5) * hh * hh, w3 = 0.5 * (x3 - 2.0 * x4 + x5) * hh * hh;
        const double d0 = (-30.0 * x2 + 60.0 * x3 - 30.0 * x4) / hh, d5 = -d0;
        const double d1 = 1.0 - 18.0 * x2 + 32.0 * x3 - 15.0 * x4, d4 = -12.0 * x2 + 28.0 * x3 - 15.0 * x4;
        const double d2 = 0.5 * (2.0 * x - 9.0 * x2 + 12.0 * x3 - 5.0 * x4) * hh, d3 = 0.5 * (3.0 * x2 - 8.0 * x3 + 5.0 * x4) * hh;
        const size_t o = (size_t)r * F + f;
        a.z[o] = fma(w0, z0, fma(w5, z1, fma(w1, v0, fma(w4, v1, fma(w2, a0, w3 * a1)))));
        a.zt[o] = fma(d0, z0, fma(d5, z1, fma(d1, v0, fma(d4, v1, fma(d2, a0, d3 * a1)))));
        if (a.slope) {
            const float g0 = (float)(2.0 * x3 - 3.0 * x2 + 1.0), g1 = (float)((x3 - 2.0 * x2 + x) * hh),
                        g2 = (float)((x3 - x2) * hh), g3 = (float)(-2.0 * x3 + 3.0 * x2);
            a.slope[o] = make_float2(fmaf(g0, s0.x, fmaf(g1, r0.x, fmaf(g2, r1.x, g3 * s1.x))),
                                     fmaf(g0, s0.y, fmaf(g1, r0.y, fmaf(g2, r1.y, g3 * s1.y))));
        }
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

cudaError_t launch_surface_refine(const SurfaceRefineArgs &a, cudaStream_t s)
{
    if (a.n_rows <= 0) return cudaSuccess;
    surface_refine_kernel<<<(unsigned)((a.n_facets + 255) / 256), 256, 0, s>>>(a);
    return cudaGetLastError();
}

cudaError_t launch_surface_slope(const DevParams &prm, const SurfaceArgs &sa, const PulseConst *pulses, int p,
                                 float2 *out, cudaStream_t s)
{
    const size_t F = (size_t)prm.nx * prm.ny;
    surface_slope_kernel<<<(unsigned)((F + 255) / 256), 256, 0, s>>>(prm, sa, pulses, p, out);
    return cudaGetLastError();
}

// Row slots a launch of the second-derivative (coarse keyframe) rows pays for: blocks of four rows, or of three when
// that wastes none (a block's spare rows recompute its last one).
int kinematics_coarse_row_slots(int n_rows)
{
    const int groups = (n_rows + 3) / 4;
    return n_rows <= 3 * groups ? 3 * groups : 4 * groups;
}

cudaError_t launch_kinematics(const DevParams &prm, const KinematicsArgs &a_in, int first, int n_rows, cudaStream_t s)
{
    if (n_rows <= 0) return cudaSuccess;
    dim3 block(kBX, kBY);
    // rows split evenly over the fewest blocks of <= kPK rows (17 rows -> 6 + 6 + 5, not 8 + 8 + 1); at least 4 rows
    // per block (a shorter launch recomputes its last row)
    const int n_chunks = (n_rows + kPK - 1) / kPK, nk = std::max(4, (n_rows + n_chunks - 1) / n_chunks);
    dim3 grid((prm.ny + kBY * kNF - 1) / (kBY * kNF), (prm.nx + kBX - 1) / kBX, (n_rows + nk - 1) / nk);   // (j blocks, i blocks, rows)
    KinematicsArgs a = a_in;
    if (a.nodes_x > 0) {                               // one group of blocks per cell of the node lattice
        const int cell_facets = (int)std::ceil(a.node_spacing / prm.spacing) + 1;
        a.chunks_x = (cell_facets + kBX - 1) / kBX; a.chunks_y = (cell_facets + kBY * kNF - 1) / (kBY * kNF);
        grid.y = (a.nodes_x - 1) * a.chunks_x; grid.x = (a.nodes_y - 1) * a.chunks_y;
    }
    const bool slope = a.slope != nullptr, choppy = a.dxy != nullptr, rate = a.H > 1;
    auto launch = [&](auto kern) { kern<<<grid, block, 0, s>>>(prm, a, first, n_rows); };
    if (a.ztt) {                                       // second-derivative rows: 4 rows per block (register budget), no CWM
        if (!rate || choppy || (slope && !a.slope_t)) return cudaErrorInvalidValue;
        grid.z = (n_rows + 3) / 4;
        if (kinematics_coarse_row_slots(n_rows) == 3 * (int)grid.z) {   // <= 3, 5, 6 or 9 rows: blocks of three (fewer rows computed twice)
            grid.z = (n_rows + 2) / 3;
            if (a.nodes_x > 0) {
                if (slope) launch(kinematics_kernel<3, true, false, true, true, true>);
                else       launch(kinematics_kernel<3, false, false, true, true, true>);
            } else {
                if (slope) launch(kinematics_kernel<3, true, false, true, false, true>);
                else       launch(kinematics_kernel<3, false, false, true, false, true>);
            }
        } else if (a.nodes_x > 0) {
            if (slope) launch(kinematics_kernel<4, true, false, true, true, true>);
            else       launch(kinematics_kernel<4, false, false, true, true, true>);
        } else {
            if (slope) launch(kinematics_kernel<4, true, false, true, false, true>);
            else       launch(kinematics_kernel<4, false, false, true, false, true>);
        }
        return cudaGetLastError();
    }
    auto pick2 = [&](auto nk_tag, auto het_tag) {
        constexpr int NK = decltype(nk_tag)::value;
        constexpr bool HET = decltype(het_tag)::value;
        if (rate) {
            if (slope && choppy) launch(kinematics_kernel<NK, true, true, true, HET>);
            else if (slope)      launch(kinematics_kernel<NK, true, false, true, HET>);
            else if (choppy)     launch(kinematics_kernel<NK, false, true, true, HET>);
            else                 launch(kinematics_kernel<NK, false, false, true, HET>);
        } else {
            if (slope && choppy) launch(kinematics_kernel<NK, true, true, false, HET>);
            else if (slope)      launch(kinematics_kernel<NK, true, false, false, HET>);
            else if (choppy)     launch(kinematics_kernel<NK, false, true, false, HET>);
            else                 launch(kinematics_kernel<NK, false, false, false, HET>);
        }
    };
    auto pick = [&](auto nk_tag) {
        if (a.nodes_x > 0) pick2(nk_tag, std::true_type{});
        else pick2(nk_tag, std::false_type{});
    };
    switch (nk) {
        case 4: pick(std::integral_constant<int, 4>{}); break;
        case 5: pick(std::integral_constant<int, 5>{}); break;
        default: pick(std::integral_constant<int, 6>{}); break;
    }
    return cudaGetLastError();
}

}  // namespace heeps
