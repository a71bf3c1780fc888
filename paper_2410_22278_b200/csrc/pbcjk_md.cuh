// McMurchie-Davidson building blocks for the real-space (erfc) quartet kernels.
//   Boys F_m: tabulated Taylor coefficients + downward recursion (eq 28 L209 is m = 0; split eq 30)
//   merged base values R^m_000 = (-2 alpha)^m F_m(alpha r^2) - theta (-2 alpha_w)^m F_m(alpha_w r^2)
//     (eq 50 L362 applied to both terms of eq 56; merged BEFORE the recursion because eq 47-49
//      depend only on the separation vector)
//   Hermite Coulomb integrals R^0_tuv by eq 47-49 (L354-360), in place
//   Hermite expansion coefficients E^{ij}_t by eq 17-20 (L138-147), with E^{00}_0 = 1 (eq 19's
//     Gaussian lives in the pair coefficient)
#pragma once
#include "pbcjk_common.h"

namespace pbcjk {

// Boys tables (built on the host at create, pbcjk_api.cu):
//   c  [LTOT+1][BOYS_ROWS][8]: Taylor coefficients of F_L around the grid point x_i = i*BOYS_DX,
//        c[L][i][k] = F_{L+k}(x_i)/k!   (d/dx F_m = -F_{m+1}), so F_L(x) = sum_k c_k (x_i - x)^k   (Horner, 7 FMA);
//        one row = one 64-byte line, read as four 16-byte loads
//   ex [BOYS_ROWS]: exp(-x_i); exp(-x) = exp(-x_i) exp(x_i - x) with a degree-8 Taylor polynomial (|x_i - x| <= 1/16:
//        truncation 4e-17) instead of a double-precision exp() call
//   cf, exf: fp32 copies for the mixed-precision evaluators
struct BoysTab {
    const double *c, *ex;
    const float *cf;
};

// F_0..F_L at x: Taylor expansion of the top order around the nearest grid point, downward recursion
// F_{m-1} = (2x F_m + e^{-x})/(2m-1); asymptotic form beyond BOYS_XMAX.
template <int L>
__device__ __forceinline__ void boys(const BoysTab &tb, double x, double *F)
{
    if (x < BOYS_XMAX) {
        const int i = __double2int_rn(x * (1.0 / BOYS_DX));
        const double dx = fma((double)i, BOYS_DX, -x);                 // x_i - x, |dx| <= 1/16
        const double2 *row = reinterpret_cast<const double2 *>(tb.c + ((size_t)L * BOYS_ROWS + i) * 8);
        const double2 c01 = __ldg(row), c23 = __ldg(row + 1), c45 = __ldg(row + 2), c67 = __ldg(row + 3);
        double f = fma(c67.y, dx, c67.x);
        f = fma(f, dx, c45.y);
        f = fma(f, dx, c45.x);
        f = fma(f, dx, c23.y);
        f = fma(f, dx, c23.x);
        f = fma(f, dx, c01.y);
        f = fma(f, dx, c01.x);
        F[L] = f;
        if (L > 0) {
            double e = fma(1.0 / 40320.0, dx, 1.0 / 5040.0);
            e = fma(e, dx, 1.0 / 720.0);
            e = fma(e, dx, 1.0 / 120.0);
            e = fma(e, dx, 1.0 / 24.0);
            e = fma(e, dx, 1.0 / 6.0);
            e = fma(e, dx, 0.5);
            e = fma(e, dx, 1.0);
            e = fma(e, dx, 1.0);
            const double ex = __ldg(tb.ex + i) * e;
            const double x2 = x + x;
#pragma unroll
            for (int m = L; m > 0; --m) F[m - 1] = fma(x2, F[m], ex) * (1.0 / (2.0 * m - 1.0));
        }
    } else {
        // F_0 = sqrt(pi/x)/2 up to e^-x (< 3e-16 here); F_{m+1} = (2m+1) F_m / (2x)
        const double rs = rsqrt(x);
        const double ix = rs * rs;
        F[0] = 0.88622692545275801365 * rs;
#pragma unroll
        for (int m = 0; m < L; ++m) F[m + 1] = F[m] * ((m + 0.5) * ix);
    }
}

// fp32 variant (mixed precision, PAPER 3.5 L817): degree-5 Taylor (|dx|^6/720 < 1e-10), fast exp
template <int L>
__device__ __forceinline__ void boys(const BoysTab &tb, float x, float *F)
{
    if (x < (float)BOYS_XMAX) {
        const int i = __float2int_rn(x * (float)(1.0 / BOYS_DX));
        const float dx = fmaf((float)i, (float)BOYS_DX, -x);
        const float4 *row = reinterpret_cast<const float4 *>(tb.cf + ((size_t)L * BOYS_ROWS + i) * 8);
        const float4 c03 = __ldg(row), c47 = __ldg(row + 1);
        float f = fmaf(c47.y, dx, c47.x);
        f = fmaf(f, dx, c03.w);
        f = fmaf(f, dx, c03.z);
        f = fmaf(f, dx, c03.y);
        f = fmaf(f, dx, c03.x);
        F[L] = f;
        if (L > 0) {
            const float ex = __expf(-x);
            const float x2 = x + x;
#pragma unroll
            for (int m = L; m > 0; --m) F[m - 1] = fmaf(x2, F[m], ex) * (1.0f / (2.0f * m - 1.0f));
        }
    } else {
        const float rs = rsqrtf(x);
        const float ix = rs * rs;
        F[0] = 0.886226925f * rs;
#pragma unroll
        for (int m = 0; m < L; ++m) F[m + 1] = F[m] * ((m + 0.5f) * ix);
    }
}

// Rm[m] = pref * [ (-2 alpha)^m F_m(alpha r2) - theta (-2 alpha_w)^m F_m(alpha_w r2) ],  m = 0..L
template <int L, typename T>
__device__ __forceinline__ void boys_merged(const BoysTab &tb, T r2, T alpha, T alpha_w, T theta, T pref, T *Rm)
{
    T F1[L + 1], F2[L + 1];
    boys<L>(tb, alpha * r2, F1);
    boys<L>(tb, alpha_w * r2, F2);
    T c1 = pref, c2 = -pref * theta;
    const T m2a = T(-2.0) * alpha, m2w = T(-2.0) * alpha_w;
#pragma unroll
    for (int m = 0; m <= L; ++m) {
        Rm[m] = fma(c1, F1[m], c2 * F2[m]);
        c1 *= m2a;
        c2 *= m2w;
    }
}

// R[hidx(t,u,v)] = R^0_tuv for t+u+v <= L, from Rm[m] = R^m_000.  In place: after the pass for level
// m the array holds R^m_tuv for t+u+v <= L-m.  Orders are visited downwards inside a level so that
// the (m+1)-level values of order n-1, n-2 are still there when order n is formed.
template <int L>
__device__ __forceinline__ void hermite_R(double *R, const double *Rm, double X, double Y, double Z)
{
    R[0] = Rm[L];
#pragma unroll
    for (int m = L - 1; m >= 0; --m) {
#pragma unroll
        for (int n = L - m; n >= 1; --n) {
#pragma unroll
            for (int t = n; t >= 0; --t) {
#pragma unroll
                for (int u = n - t; u >= 0; --u) {
                    const int v = n - t - u;
                    double val;
                    if (t > 0) {                                          // eq 47
                        val = X * R[hidx(t - 1, u, v)];
                        if (t > 1) val = fma((double)(t - 1), R[hidx(t - 2, u, v)], val);
                    } else if (u > 0) {                                   // eq 48
                        val = Y * R[hidx(t, u - 1, v)];
                        if (u > 1) val = fma((double)(u - 1), R[hidx(t, u - 2, v)], val);
                    } else {                                              // eq 49
                        val = Z * R[hidx(t, u, v - 1)];
                        if (v > 1) val = fma((double)(v - 1), R[hidx(t, u, v - 2)], val);
                    }
                    R[hidx(t, u, v)] = val;
                }
            }
        }
        R[0] = Rm[m];
    }
}

// One Cartesian direction of the Hermite expansion coefficients (eq 17-18), E^{00}_0 = 1.
template <int LA, int LB>
struct E1D {
    double e[LA + 1][LB + 1][LA + LB + 1];
    __device__ __forceinline__ void build(double PA, double PB, double o2p)
    {
#pragma unroll
        for (int i = 0; i <= LA; ++i)
#pragma unroll
            for (int j = 0; j <= LB; ++j)
#pragma unroll
                for (int t = 0; t <= LA + LB; ++t) e[i][j][t] = 0.0;
        e[0][0][0] = 1.0;
#pragma unroll
        for (int i = 0; i < LA; ++i)
#pragma unroll
            for (int t = 0; t <= i + 1; ++t) {
                double v = 0.0;
                if (t <= i) v = PA * e[i][0][t];
                if (t > 0) v = fma(o2p, e[i][0][t - 1], v);
                if (t + 1 <= i) v = fma((double)(t + 1), e[i][0][t + 1], v);
                e[i + 1][0][t] = v;
            }
#pragma unroll
        for (int i = 0; i <= LA; ++i)
#pragma unroll
            for (int j = 0; j < LB; ++j)
#pragma unroll
                for (int t = 0; t <= i + j + 1; ++t) {
                    double v = 0.0;
                    if (t <= i + j) v = PB * e[i][j][t];
                    if (t > 0) v = fma(o2p, e[i][j][t - 1], v);
                    if (t + 1 <= i + j) v = fma((double)(t + 1), e[i][j][t + 1], v);
                    e[i][j + 1][t] = v;
                }
    }
};

// Cartesian powers of component k of a shell with angular momentum l <= 2 (order x,y,z / xx,xy,xz,yy,yz,zz:
// PAPER L721).  Closed forms, so that they fold to constants as soon as k is one (unrolled loops).
__host__ __device__ constexpr int cart_x(int l, int k)
{
    return l == 0 ? 0 : (l == 1 ? (k == 0 ? 1 : 0) : (k == 0 ? 2 : (k < 3 ? 1 : 0)));
}
__host__ __device__ constexpr int cart_y(int l, int k)
{
    return l == 0 ? 0 : (l == 1 ? (k == 1 ? 1 : 0) : (k == 3 ? 2 : ((k == 1 || k == 4) ? 1 : 0)));
}
__host__ __device__ constexpr int cart_z(int l, int k) { return l - cart_x(l, k) - cart_y(l, k); }

// runtime-l variant used by the light kernels (density prep, J back-transform, rho(G) generation)
struct E1Drt {
    double e[LMAX + 1][LMAX + 1][2 * LMAX + 1];
    __device__ void build(int la, int lb, double PA, double PB, double o2p)
    {
        for (int i = 0; i <= LMAX; ++i)
            for (int j = 0; j <= LMAX; ++j)
                for (int t = 0; t <= 2 * LMAX; ++t) e[i][j][t] = 0.0;
        e[0][0][0] = 1.0;
        for (int i = 0; i < la; ++i)
            for (int t = 0; t <= i + 1; ++t) {
                double v = 0.0;
                if (t <= i) v = PA * e[i][0][t];
                if (t > 0) v += o2p * e[i][0][t - 1];
                if (t + 1 <= i) v += (t + 1) * e[i][0][t + 1];
                e[i + 1][0][t] = v;
            }
        for (int i = 0; i <= la; ++i)
            for (int j = 0; j < lb; ++j)
                for (int t = 0; t <= i + j + 1; ++t) {
                    double v = 0.0;
                    if (t <= i + j) v = PB * e[i][j][t];
                    if (t > 0) v += o2p * e[i][j][t - 1];
                    if (t + 1 <= i + j) v += (t + 1) * e[i][j][t + 1];
                    e[i][j + 1][t] = v;
                }
    }
};

__device__ __forceinline__ void cart_powers(int l, int k, int &x, int &y, int &z)
{
    // l <= 2
    if (l == 0) { x = y = z = 0; }
    else if (l == 1) { x = (k == 0); y = (k == 1); z = (k == 2); }
    else {
        const int tx[6] = {2, 1, 1, 0, 0, 0}, ty[6] = {0, 1, 0, 2, 1, 0};
        x = tx[k]; y = ty[k]; z = 2 - x - y;
    }
}

}  // namespace pbcjk
