// blip_f64.cuh — fp64 evaluation kernel (product path).
//
// The paper keeps the local-energy evaluation in double precision on the CPU because the bias
// of single-precision orbitals in the energy is untested and uses the fp32 GPU
// values only for accept/reject.  This kernel is the same evaluation (Eq. 6-8)
// with fp64 weights, fp64 accumulation and fp64 outputs from the same resident fp32 table, so
// that the occasional local-energy call can stay on the device too.  It is the accuracy path,
// not the fast one: same layout as the split kernel (CTA = electron x 128 orbitals, warp m1 =
// the 16 rows of plane i1 + m1, partial sums added in plane order), no grouping.
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
