// McMurchie-Davidson building blocks for the real-space (erfc) quartet kernels.
//   Boys F_m: tabulated, Taylor + downward recursion (eq 28 L209 is m = 0; split eq 30)
//   merged base values R^m_000 = (-2 alpha)^m F_m(alpha r^2) - theta (-2 alpha_w)^m F_m(alpha_w r^2)
//     (eq 50 L362 applied to both terms of eq 56; merged BEFORE the recursion because eq 47-49
//      depend only on the separation vector)
//   Hermite Coulomb integrals R^0_tuv by eq 47-49 (L354-360), in place
//   Hermite expansion coefficients E^{ij}_t by eq 17-20 (L138-147), with E^{00}_0 = 1 (eq 19's
//     Gaussian lives in the pair coefficient)
#pragma once
#include "pbcjk_common.h"

namespace pbcjk {

// F_0..F_L at x.  tab: BOYS_ROWS x BOYS_MCOL, tab[i][m] = F_m(i*BOYS_DX).
template <int L>
__device__ __forceinline__ void boys(const double *__restrict__ tab, double x, double *F)
{
    if (x < BOYS_XMAX) {
        int i = __double2int_rn(x * (1.0 / BOYS_DX));
        double dx = fma((double)i, BOYS_DX, -x);                 // x0 - x, |dx| <= 1/16
        const double *row = tab + i * BOYS_MCOL + L;
        // F_L(x) = sum_k F_{L+k}(x0) dx^k / k!   (d/dx F_m = -F_{m+1}), nested form
        double f = __ldg(row + 7);
        f = fma(f, dx * (1.0 / 7.0), __ldg(row + 6));
        f = fma(f, dx * (1.0 / 6.0), __ldg(row + 5));
        f = fma(f, dx * (1.0 / 5.0), __ldg(row + 4));
        f = fma(f, dx * (1.0 / 4.0), __ldg(row + 3));
        f = fma(f, dx * (1.0 / 3.0), __ldg(row + 2));
        f = fma(f, dx * 0.5, __ldg(row + 1));
        f = fma(f, dx, __ldg(row));
        F[L] = f;
        if (L > 0) {
            double ex = exp(-x);
            double x2 = x + x;
#pragma unroll
            for (int m = L; m > 0; --m) F[m - 1] = fma(x2, F[m], ex) * (1.0 / (2.0 * m - 1.0));
        }
    } else {
        // F_0 = sqrt(pi/x)/2 up to e^-x (< 3e-16 here); F_{m+1} = (2m+1) F_m / (2x)
        double rs = rsqrt(x);
        double ix = rs * rs;
        F[0] = 0.88622692545275801365 * rs;
#pragma unroll
        for (int m = 0; m < L; ++m) F[m + 1] = F[m] * ((m + 0.5) * ix);
    }
}

// Rm[m] = pref * [ (-2 alpha)^m F_m(alpha r2) - theta (-2 alpha_w)^m F_m(alpha_w r2) ],  m = 0..L
template <int L>
__device__ __forceinline__ void boys_merged(const double *__restrict__ tab, double r2, double alpha,
                                            double alpha_w, double theta, double pref, double *Rm)
{
    double F1[L + 1], F2[L + 1];
    boys<L>(tab, alpha * r2, F1);
    boys<L>(tab, alpha_w * r2, F2);
    double c1 = pref, c2 = -pref * theta;
    double m2a = -2.0 * alpha, m2w = -2.0 * alpha_w;
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
