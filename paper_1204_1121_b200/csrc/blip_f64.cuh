// blip_f64.cuh — the accuracy / Hessian kernel (product path).
//
// The paper keeps the local-energy evaluation in double precision on the CPU because the bias
// of single-precision orbitals in the energy is untested and uses the fp32 GPU
// values only for accept/reject; the local-energy call is also the one that needs second
// derivatives.  eval_full_kernel<T, MODE> is the same evaluation (Eq. 6-8,
// PAPER.md:78-102) from the same resident fp32 table with
//     T = double            fp64 fraction, weights, accumulation and outputs (blipgpu_eval_f64)
//     MODE 0 / 1 / 2        value / value + gradient + Laplacian / value + gradient + the full
//                           Cartesian Hessian (6 components: xx yy zz xy xz yz), T = float or double
// so that the occasional local-energy call can stay on the device too.  It is the accuracy
// path, not the fast one: same layout as the split kernel (CTA = electron x 128 orbitals, warp
// m1 = the 16 rows of plane i1 + m1, all in flight at once while the weights are computed, partial
// sums added in plane order), no grouping.
//
// Arithmetic, z axis contracted first as in blip_kernels.cuh: per column (m1, m2)
//     a = sum_m3 w3 c,  b = sum_m3 w3' c,  d = sum_m3 w3'' c        (MODE 1: d carries Q22)
// MODE 1 folds them into {S, T1, T2, T3, lap} with {P00, P10, P01, La, Lb} (ElecRec comment);
// MODE 2 keeps all ten grid-space sums
//     S += P00 a   T1 += P10 a   T2 += P01 a   T3 += P00 b
//     H11 += P20 a   H22 += P02 a   H33 += P00 d   H12 += P11 a   H13 += P10 b   H23 += P01 b
// (P20 = w1'' w2, P02 = w1 w2'', P11 = w1' w2') and maps them once per orbital:
//     grad_i = sum_a J[a][i] T_a,    Hc[i][j] = sum_ab J[a][i] H_ab J[b][j]      (t = J r, J constant).
#pragma once
#include "blip_kernels.cuh"

namespace blip {

// cell map of one axis with the fraction kept in fp64 (same pinned sequence as cell_map_axis)
__device__ __forceinline__ bool cell_map_axis_d(const Geom& g, int a, double x, double y, double z,
                                                int& i, double& f)
{
    double u = __dadd_rn(__dadd_rn(__dmul_rn(x, g.G[a]), __dmul_rn(y, g.G[3 + a])),
                         __dmul_rn(z, g.G[6 + a]));
    if (!isfinite(u)) { i = -1; f = 0.0; return false; }
    u = __dsub_rn(u, floor(u));
    double t = __dmul_rn(u, (double)g.n[a]);
    int ia = (int)floor(t);
    if (ia >= g.n[a]) { ia -= g.n[a]; t = __dsub_rn(t, (double)g.n[a]); }
    i = ia;
    f = __dsub_rn(t, (double)ia);
    return true;
}

// the 1-D factor and its derivatives at site m (see phi_site), in T
template <typename T>
__device__ __forceinline__ void phi_site_t(T f, int m, T& w, T& d1, T& d2)
{
    const bool mirrored = (m == 0) || (m == 2);
    const T x = mirrored ? T(1) - f : f;
    const T sg = mirrored ? T(-1) : T(1);
    const T x2 = x * x;
    if (m == 0 || m == 3) {
        w = x2 * x * (T(1) / T(6));
        d1 = sg * T(0.5) * x2;
        d2 = x;
    } else {
        w = T(2) / T(3) - x2 * (T(1) - T(0.5) * x);
        d1 = sg * x * (T(1.5) * x - T(2));
        d2 = T(3) * x - T(2);
    }
}

template <int MODE> struct FullShape {
    static constexpr int NCW = MODE == 2 ? 6 : 5;           // per-column weights
    static constexpr int NACC = MODE == 0 ? 1 : (MODE == 1 ? 5 : 10);
};

// per-electron record of the kernel (same content as ElecRec, in T)
template <typename T, int MODE>
struct FullRec {
    T cw[16][6];        // column (m1,m2): MODE 1 {P00, P10, P01, La, Lb, -}; MODE 2 {P00, P10, P01, P20, P02, P11}
    T wz[3][4];         // w3, w3', w3'' (MODE 1: Q22 w3'')
    T ax[3][3][4];      // scratch: per-axis factors
};

// one column (m1, m2) of one orbital: c[0..3] the coefficients of the 4 z sites
template <typename T, int MODE>
__device__ __forceinline__ void fold_full(const float (&c)[4], const FullRec<T, MODE>& r, int col, T (&acc)[FullShape<MODE>::NACC])
{
    const T c0 = c[0], c1 = c[1], c2 = c[2], c3 = c[3];
    const T* w = r.cw[col];
    const T a = fma(c3, r.wz[0][3], fma(c2, r.wz[0][2], fma(c1, r.wz[0][1], c0 * r.wz[0][0])));
    acc[0] = fma(a, w[0], acc[0]);
    if (MODE != 0) {
        const T b = fma(c3, r.wz[1][3], fma(c2, r.wz[1][2], fma(c1, r.wz[1][1], c0 * r.wz[1][0])));
        const T d = fma(c3, r.wz[2][3], fma(c2, r.wz[2][2], fma(c1, r.wz[2][1], c0 * r.wz[2][0])));
        acc[1] = fma(a, w[1], acc[1]);
        acc[2] = fma(a, w[2], acc[2]);
        acc[3] = fma(b, w[0], acc[3]);
        if (MODE == 1) {
            acc[4] = fma(d, w[0], fma(b, w[4], fma(a, w[3], acc[4])));
        } else {
            acc[4] = fma(a, w[3], acc[4]);                   // H11
            acc[5] = fma(a, w[4], acc[5]);                   // H22
            acc[6] = fma(d, w[0], acc[6]);                   // H33
            acc[7] = fma(a, w[5], acc[7]);                   // H12
            acc[8] = fma(b, w[1], acc[8]);                   // H13
            acc[9] = fma(b, w[2], acc[9]);                   // H23
        }
    }
}

__device__ __forceinline__ void st_stream_quad(double* p, double a, double b, double c, double d)
{
    asm volatile("st.global.cs.v2.f64 [%0], {%1, %2};" :: "l"(p), "d"(a), "d"(b) : "memory");
    asm volatile("st.global.cs.v2.f64 [%0], {%1, %2};" :: "l"(p + 2), "d"(c), "d"(d) : "memory");
}
__device__ __forceinline__ void st_stream_quad(float* p, float a, float b, float c, float d)
{
    st_stream4(p, a, b, c, d);
}

// grid (M, ceil(L / 128)), block 128.  Outputs in T: val [M][ld], grad [M][3][ld] (MODE >= 1),
// third [M][ld] = Laplacian (MODE 1) or [M][6][ld] = Hessian xx yy zz xy xz yz (MODE 2).
template <typename T, int MODE>
__global__ void __launch_bounds__(128, sizeof(T) == 8 ? 3 : 1)      // fp64: at most 168 registers, 12 warps per SM
eval_full_kernel(Geom g, Geom64 g64, const float4* __restrict__ table4, const double* __restrict__ pos, long long M,
                 T* __restrict__ val, T* __restrict__ grad, T* __restrict__ third, long long ld,
                 int* __restrict__ cell_out)
{
    constexpr int NACC = FullShape<MODE>::NACC;
    __shared__ FullRec<T, MODE> recw[4];                     // one per warp
    __shared__ T part[3][4 * NACC][32];                      // partial sums of warps 1..3: [orbital j][quantity][lane]
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int e = blockIdx.x;
    const int quad = blockIdx.y * 32 + lane;
    FullRec<T, MODE>& rec = recw[warp];
    // a-1 by every warp (lanes 0..11 = axis lane / 4, site lane % 4), then its 16 loads at once,
    // then the weights while the loads are in flight (as eval_split_kernel)
    const double x = pos[3 * (size_t)e], y = pos[3 * (size_t)e + 1], z = pos[3 * (size_t)e + 2];
    int ia = 0; double fa = 0.0;
    if (lane < 12) cell_map_axis_d(g, lane >> 2, x, y, z, ia, fa);
    const int i1 = __shfl_sync(0xffffffffu, ia, 0), i2 = __shfl_sync(0xffffffffu, ia, 4), i3 = __shfl_sync(0xffffffffu, ia, 8);
    const bool ok = (i1 | i2 | i3) >= 0;
    if (cell_out && blockIdx.y == 0 && warp == 0 && lane < 12 && (lane & 3) == 0) cell_out[3 * (size_t)e + (lane >> 2)] = ok ? ia : -1;
    float4 buf[4][4];
    // fp32: the 16 loads go out first and the weights are computed under them.  fp64: holding 64
    // loaded registers across the weight code costs more (occupancy) than it hides, so they follow it
    constexpr bool kLoadsFirst = sizeof(T) == 4;
    auto issue_loads = [&]() {
        if (!ok) return;
        const unsigned off = (unsigned)min(quad, g.pitch4 - 1);
        const unsigned s2 = (unsigned)g.np[2];
        const unsigned row0 = ((unsigned)(i1 + warp) * g.np[1] + i2) * g.np[2] + i3;
#pragma unroll
        for (int m2 = 0; m2 < 4; ++m2)
#pragma unroll
            for (int m3 = 0; m3 < 4; ++m3)
                buf[m2][m3] = __ldg(table4 + ((size_t)(row0 + m2 * s2 + m3) * (size_t)g.pitch4 + off));
    };
    if (kLoadsFirst) issue_loads();
    if (lane < 12) {
        const int a = lane >> 2, m = lane & 3;
        phi_site_t<T>((T)fa, m, rec.ax[a][0][m], rec.ax[a][1][m], rec.ax[a][2][m]);
    }
    __syncwarp();
    if (lane < 16) {
        const int m1 = lane >> 2, m2 = lane & 3;
        const T a0 = rec.ax[0][0][m1], b0 = rec.ax[0][1][m1], c0 = rec.ax[0][2][m1];
        const T a1 = rec.ax[1][0][m2], b1 = rec.ax[1][1][m2], c1 = rec.ax[1][2][m2];
        const T p00 = a0 * a1, p10 = b0 * a1, p01 = a0 * b1;
        rec.cw[lane][0] = p00; rec.cw[lane][1] = p10; rec.cw[lane][2] = p01;
        if (MODE == 2) {
            rec.cw[lane][3] = c0 * a1; rec.cw[lane][4] = a0 * c1; rec.cw[lane][5] = b0 * b1;
        } else {
            rec.cw[lane][3] = (T)g64.Q[0] * c0 * a1 + (T)g64.Q[1] * a0 * c1 + T(2) * (T)g64.Q[3] * b0 * b1;
            rec.cw[lane][4] = T(2) * ((T)g64.Q[4] * p10 + (T)g64.Q[5] * p01);
            rec.cw[lane][5] = T(0);
        }
    } else if (lane < 28) {
        const int k = (lane - 16) >> 2, m = lane & 3;
        rec.wz[k][m] = (k == 2 && MODE == 1) ? (T)g64.Q[2] * rec.ax[2][2][m] : rec.ax[2][k][m];
    }
    __syncwarp();
    if (!kLoadsFirst) issue_loads();

    T acc[4][NACC];
#pragma unroll
    for (int j = 0; j < 4; ++j)
#pragma unroll
        for (int q = 0; q < NACC; ++q) acc[j][q] = T(0);
    if (ok) {
#pragma unroll
        for (int m2 = 0; m2 < 4; ++m2) {
            const int col = 4 * warp + m2;
            const float cx[4] = {buf[m2][0].x, buf[m2][1].x, buf[m2][2].x, buf[m2][3].x};
            const float cy[4] = {buf[m2][0].y, buf[m2][1].y, buf[m2][2].y, buf[m2][3].y};
            const float cz[4] = {buf[m2][0].z, buf[m2][1].z, buf[m2][2].z, buf[m2][3].z};
            const float cq[4] = {buf[m2][0].w, buf[m2][1].w, buf[m2][2].w, buf[m2][3].w};
            fold_full<T, MODE>(cx, rec, col, acc[0]); fold_full<T, MODE>(cy, rec, col, acc[1]);
            fold_full<T, MODE>(cz, rec, col, acc[2]); fold_full<T, MODE>(cq, rec, col, acc[3]);
        }
    }
    if (warp > 0) {
#pragma unroll
        for (int j = 0; j < 4; ++j)
#pragma unroll
            for (int q = 0; q < NACC; ++q) part[warp - 1][NACC * j + q][lane] = acc[j][q];
    }
    __syncthreads();
    if (warp != 0 || quad >= g.pitch4) return;
    const T nan = (T)__longlong_as_double(0x7ff8000000000000ll);
    T J[9];
#pragma unroll
    for (int k = 0; k < 9; ++k) J[k] = (T)g64.J[k];
    T v[4], gr[3][4], th[6][4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        T s[NACC];
#pragma unroll
        for (int q = 0; q < NACC; ++q) {
            s[q] = acc[j][q];
#pragma unroll
            for (int w = 0; w < 3; ++w) s[q] += part[w][NACC * j + q][lane];
        }
        v[j] = ok ? s[0] : nan;
        if (MODE != 0) {
#pragma unroll
            for (int i = 0; i < 3; ++i) gr[i][j] = ok ? J[i] * s[1] + J[3 + i] * s[2] + J[6 + i] * s[3] : nan;
        }
        if (MODE == 1) th[0][j] = ok ? s[4] : nan;
        if (MODE == 2) {
            // grid-space Hessian, symmetric: Ht[a][b]
            const T Ht[3][3] = {{s[4], s[7], s[8]}, {s[7], s[5], s[9]}, {s[8], s[9], s[6]}};
            const int ci[6] = {0, 1, 2, 0, 0, 1}, cj[6] = {0, 1, 2, 1, 2, 2};
#pragma unroll
            for (int q = 0; q < 6; ++q) {
                T h = T(0);
#pragma unroll
                for (int a = 0; a < 3; ++a) {
                    const T row = Ht[a][0] * J[cj[q]] + Ht[a][1] * J[3 + cj[q]] + Ht[a][2] * J[6 + cj[q]];   // sum_b Ht[a][b] J[b][j]
                    h = fma(J[3 * a + ci[q]], row, h);
                }
                th[q][j] = ok ? h : nan;
            }
        }
    }
    const size_t o = (size_t)e * (size_t)ld + 4 * (size_t)quad;
    st_stream_quad(val + o, v[0], v[1], v[2], v[3]);
    if (MODE != 0) {
        const size_t og = (size_t)e * 3 * (size_t)ld + 4 * (size_t)quad;
#pragma unroll
        for (int i = 0; i < 3; ++i) st_stream_quad(grad + og + i * ld, gr[i][0], gr[i][1], gr[i][2], gr[i][3]);
    }
    if (MODE == 1) st_stream_quad(third + o, th[0][0], th[0][1], th[0][2], th[0][3]);
    if (MODE == 2) {
        const size_t oh = (size_t)e * 6 * (size_t)ld + 4 * (size_t)quad;
#pragma unroll
        for (int q = 0; q < 6; ++q) st_stream_quad(third + oh + q * ld, th[q][0], th[q][1], th[q][2], th[q][3]);
    }
}

// ---------------------------------------------------------------------------------------
// fp64 value / value + gradient + Laplacian (blipgpu_eval_f64, modes VALUE and VGL): the kernel
// of round 1, kept as it was — one record per CTA prepared by warp 0, 128 registers, 16 warps per
// SM.  The generic eval_full_kernel<double, 1> computes the same numbers but runs 20-60 % slower
// (its per-warp preparation keeps the 64 loaded registers live across the weight code: 224
// registers, 8 warps per SM), so it serves the Hessian mode and the fp32 Hessian only.
// ---------------------------------------------------------------------------------------
// the 1-D factor and its derivatives at site m (see phi_site), in fp64
__device__ __forceinline__ void phi_site_d(double f, int m, double& w, double& d1, double& d2)
{
    const bool mirrored = (m == 0) || (m == 2);
    const double x = mirrored ? 1.0 - f : f;
    const double sg = mirrored ? -1.0 : 1.0;
    const double x2 = x * x;
    if (m == 0 || m == 3) {
        w = x2 * x * (1.0 / 6.0);
        d1 = sg * 0.5 * x2;
        d2 = x;
    } else {
        w = 2.0 / 3.0 - x2 * (1.0 - 0.5 * x);
        d1 = sg * x * (1.5 * x - 2.0);
        d2 = 3.0 * x - 2.0;
    }
}

// per-electron record of the fp64 kernel (same content as ElecRec, in doubles)
struct ElecRec64 {
    double cw[16][4];   // column (m1,m2): {P00, P10, P01, La}
    double lb[16];      // column: Lb
    double wz[3][4];    // w3, w3', Q22 w3''
    double ax[3][3][4]; // scratch: per-axis factors
    int    i[3];
    int    ok;
};

struct Acc64 { double val, t1, t2, t3, lp; };

// one column (m1, m2) of one orbital: c[0..3] the coefficients of the 4 z sites
template <int MODE>
__device__ __forceinline__ void fold64(const float (&c)[4], const ElecRec64& r, int col, Acc64& acc)
{
    const double c0 = c[0], c1 = c[1], c2 = c[2], c3 = c[3];
    const double a = fma(c3, r.wz[0][3], fma(c2, r.wz[0][2], fma(c1, r.wz[0][1], c0 * r.wz[0][0])));
    acc.val = fma(a, r.cw[col][0], acc.val);
    if (MODE != 0) {
        const double b = fma(c3, r.wz[1][3], fma(c2, r.wz[1][2], fma(c1, r.wz[1][1], c0 * r.wz[1][0])));
        const double d = fma(c3, r.wz[2][3], fma(c2, r.wz[2][2], fma(c1, r.wz[2][1], c0 * r.wz[2][0])));
        acc.t1 = fma(a, r.cw[col][1], acc.t1);
        acc.t2 = fma(a, r.cw[col][2], acc.t2);
        acc.t3 = fma(b, r.cw[col][0], acc.t3);
        acc.lp = fma(d, r.cw[col][0], fma(b, r.lb[col], fma(a, r.cw[col][3], acc.lp)));
    }
}

__device__ __forceinline__ void st_stream2d(double* p, double a, double b)
{
    asm volatile("st.global.cs.v2.f64 [%0], {%1, %2};" :: "l"(p), "d"(a), "d"(b) : "memory");
}

// grid (M, ceil(L / 128)), block 128.  Outputs fp64: val [M][ld], grad [M][3][ld], lap [M][ld].
template <int MODE>
__global__ void __launch_bounds__(128)
eval_f64_kernel(Geom g, Geom64 g64, const float4* __restrict__ table4, const double* __restrict__ pos, long long M,
                double* __restrict__ val, double* __restrict__ grad, double* __restrict__ lap, long long ld,
                int* __restrict__ cell_out)
{
    __shared__ ElecRec64 rec;
    __shared__ double part[3][4 * 5][32];                    // partial sums of warps 1..3: [orbital j][quantity][lane]
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int e = blockIdx.x;
    const int quad = blockIdx.y * 32 + lane;
    if (warp == 0) {
        const double x = pos[3 * (size_t)e], y = pos[3 * (size_t)e + 1], z = pos[3 * (size_t)e + 2];
        if (lane < 12) {
            const int a = lane >> 2, m = lane & 3;
            int ia; double fa;
            const bool ok = cell_map_axis_d(g, a, x, y, z, ia, fa);
            phi_site_d(fa, m, rec.ax[a][0][m], rec.ax[a][1][m], rec.ax[a][2][m]);
            if (m == 0) rec.i[a] = ok ? ia : -1;
        }
        __syncwarp();
        if (lane < 16) {
            const int m1 = lane >> 2, m2 = lane & 3;
            const double a0 = rec.ax[0][0][m1], b0 = rec.ax[0][1][m1], c0 = rec.ax[0][2][m1];
            const double a1 = rec.ax[1][0][m2], b1 = rec.ax[1][1][m2], c1 = rec.ax[1][2][m2];
            const double p00 = a0 * a1, p10 = b0 * a1, p01 = a0 * b1;
            rec.cw[lane][0] = p00; rec.cw[lane][1] = p10; rec.cw[lane][2] = p01;
            rec.cw[lane][3] = g64.Q[0] * c0 * a1 + g64.Q[1] * a0 * c1 + 2.0 * g64.Q[3] * b0 * b1;
            rec.lb[lane] = 2.0 * (g64.Q[4] * p10 + g64.Q[5] * p01);
        } else if (lane < 28) {
            const int k = (lane - 16) >> 2, m = lane & 3;
            rec.wz[k][m] = (k == 2) ? g64.Q[2] * rec.ax[2][2][m] : rec.ax[2][k][m];
        }
        if (lane == 0) rec.ok = (rec.i[0] | rec.i[1] | rec.i[2]) >= 0;
    }
    __syncthreads();
    const bool ok = rec.ok != 0;
    if (cell_out && blockIdx.y == 0 && threadIdx.x < 3) cell_out[3 * (size_t)e + threadIdx.x] = ok ? rec.i[threadIdx.x] : -1;

    Acc64 acc[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[j].val = acc[j].t1 = acc[j].t2 = acc[j].t3 = acc[j].lp = 0.0;
    if (ok) {
        const unsigned off = (unsigned)min(quad, g.pitch4 - 1);
        const unsigned s2 = (unsigned)g.np[2];
        const unsigned row0 = ((unsigned)(rec.i[0] + warp) * g.np[1] + rec.i[1]) * g.np[2] + rec.i[2];
        float4 buf[4][4];
#pragma unroll
        for (int m2 = 0; m2 < 4; ++m2)
#pragma unroll
            for (int m3 = 0; m3 < 4; ++m3)
                buf[m2][m3] = __ldg(table4 + ((size_t)(row0 + m2 * s2 + m3) * (size_t)g.pitch4 + off));
#pragma unroll
        for (int m2 = 0; m2 < 4; ++m2) {
            const int col = 4 * warp + m2;
            const float cx[4] = {buf[m2][0].x, buf[m2][1].x, buf[m2][2].x, buf[m2][3].x};
            const float cy[4] = {buf[m2][0].y, buf[m2][1].y, buf[m2][2].y, buf[m2][3].y};
            const float cz[4] = {buf[m2][0].z, buf[m2][1].z, buf[m2][2].z, buf[m2][3].z};
            const float cq[4] = {buf[m2][0].w, buf[m2][1].w, buf[m2][2].w, buf[m2][3].w};
            fold64<MODE>(cx, rec, col, acc[0]); fold64<MODE>(cy, rec, col, acc[1]);
            fold64<MODE>(cz, rec, col, acc[2]); fold64<MODE>(cq, rec, col, acc[3]);
        }
    }
    if (warp > 0) {
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            part[warp - 1][5 * j + 0][lane] = acc[j].val; part[warp - 1][5 * j + 1][lane] = acc[j].t1;
            part[warp - 1][5 * j + 2][lane] = acc[j].t2; part[warp - 1][5 * j + 3][lane] = acc[j].t3;
            part[warp - 1][5 * j + 4][lane] = acc[j].lp;
        }
    }
    __syncthreads();
    if (warp != 0 || quad >= g.pitch4) return;
    const double nan = __longlong_as_double(0x7ff8000000000000ll);
    double v[4], gx[4], gy[4], gz[4], lp[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        Acc64 s = acc[j];
#pragma unroll
        for (int w = 0; w < 3; ++w) {
            s.val += part[w][5 * j + 0][lane]; s.t1 += part[w][5 * j + 1][lane]; s.t2 += part[w][5 * j + 2][lane];
            s.t3 += part[w][5 * j + 3][lane]; s.lp += part[w][5 * j + 4][lane];
        }
        v[j] = ok ? s.val : nan;
        gx[j] = ok ? g64.J[0] * s.t1 + g64.J[3] * s.t2 + g64.J[6] * s.t3 : nan;
        gy[j] = ok ? g64.J[1] * s.t1 + g64.J[4] * s.t2 + g64.J[7] * s.t3 : nan;
        gz[j] = ok ? g64.J[2] * s.t1 + g64.J[5] * s.t2 + g64.J[8] * s.t3 : nan;
        lp[j] = ok ? s.lp : nan;
    }
    const size_t o = (size_t)e * (size_t)ld + 4 * (size_t)quad;
    const size_t og = (size_t)e * 3 * (size_t)ld + 4 * (size_t)quad;
    st_stream2d(val + o, v[0], v[1]); st_stream2d(val + o + 2, v[2], v[3]);
    if (MODE != 0) {
        st_stream2d(grad + og, gx[0], gx[1]); st_stream2d(grad + og + 2, gx[2], gx[3]);
        st_stream2d(grad + og + ld, gy[0], gy[1]); st_stream2d(grad + og + ld + 2, gy[2], gy[3]);
        st_stream2d(grad + og + 2 * ld, gz[0], gz[1]); st_stream2d(grad + og + 2 * ld + 2, gz[2], gz[3]);
        st_stream2d(lap + o, lp[0], lp[1]); st_stream2d(lap + o + 2, lp[2], lp[3]);
    }
}

}  // namespace blip
