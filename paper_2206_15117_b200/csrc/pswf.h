// pswf.h -- host-side evaluation of the order-zero prolate spheroidal angular function
//   psi(eta) = S00(c, eta) / S00(c, 0),  c = pi * S_ps / 2,
// the anti-aliasing function of the kernel tables ("an anti-aliasing function";
// BASELINE.json north_star: prolate-spheroidal).  Computed from its definition -- the bounded solution of
//   d/d eta [(1 - eta^2) dS/d eta] + (chi - c^2 eta^2) S = 0
// expanded in orthonormal Legendre functions, where the even-order coefficients are the eigenvector of a
// symmetric tridiagonal matrix belonging to its smallest eigenvalue.  No rational-approximation table is used.
// (The oracle evaluates the same function with scipy.special.pro_ang1: a different algorithm.)
#pragma once
#include <cmath>
#include <vector>

namespace imager {

class Pswf {
  public:
    explicit Pswf(int support) {
        const double c = M_PI * support / 2.0, c2 = c * c;
        const int K = 40;                                  // even orders r = 0, 2, ..., 2(K-1)
        std::vector<double> a(K * K, 0.0), v(K * K, 0.0);
        for (int i = 0; i < K; ++i) {
            const double r = 2.0 * i;
            a[i * K + i] = r * (r + 1) + c2 * (2 * r * (r + 1) - 1) / ((2 * r - 1) * (2 * r + 3));
            if (i + 1 < K) {
                const double off = c2 * (r + 1) * (r + 2) / ((2 * r + 3) * std::sqrt((2 * r + 1) * (2 * r + 5)));
                a[i * K + i + 1] = a[(i + 1) * K + i] = off;
            }
            v[i * K + i] = 1.0;
        }
        // cyclic Jacobi eigen-decomposition of the small symmetric matrix
        for (int sweep = 0; sweep < 60; ++sweep) {
            double off = 0;
            for (int p = 0; p < K; ++p)
                for (int q = p + 1; q < K; ++q) off += a[p * K + q] * a[p * K + q];
            if (off < 1e-300) break;
            for (int p = 0; p < K; ++p)
                for (int q = p + 1; q < K; ++q) {
                    const double apq = a[p * K + q];
                    if (std::fabs(apq) < 1e-300) continue;
                    const double theta = (a[q * K + q] - a[p * K + p]) / (2 * apq);
                    const double t = (theta >= 0 ? 1.0 : -1.0) / (std::fabs(theta) + std::sqrt(theta * theta + 1));
                    const double cs = 1 / std::sqrt(t * t + 1), sn = t * cs;
                    for (int k = 0; k < K; ++k) {
                        const double akp = a[k * K + p], akq = a[k * K + q];
                        a[k * K + p] = cs * akp - sn * akq;
                        a[k * K + q] = sn * akp + cs * akq;
                    }
                    for (int k = 0; k < K; ++k) {
                        const double apk = a[p * K + k], aqk = a[q * K + k];
                        a[p * K + k] = cs * apk - sn * aqk;
                        a[q * K + k] = sn * apk + cs * aqk;
                    }
                    for (int k = 0; k < K; ++k) {
                        const double vkp = v[k * K + p], vkq = v[k * K + q];
                        v[k * K + p] = cs * vkp - sn * vkq;
                        v[k * K + q] = sn * vkp + cs * vkq;
                    }
                }
        }
        int best = 0;
        for (int i = 1; i < K; ++i)
            if (a[i * K + i] < a[best * K + best]) best = i;
        coef_.resize(K);
        for (int i = 0; i < K; ++i) coef_[i] = v[i * K + best] * std::sqrt((4.0 * i + 1) / 2.0);   // un-normalise P_r
        norm_ = raw(0.0);
    }

    double operator()(double eta) const { return raw(eta) / norm_; }

  private:
    double raw(double x) const {
        // sum_i coef_i P_{2i}(x) with the Legendre three-term recurrence
        double pm = 1.0, p = x, s = coef_[0];
        for (int r = 1; r + 1 < 2 * (int)coef_.size(); ++r) {
            const double pn = ((2 * r + 1) * x * p - r * pm) / (r + 1);
            pm = p;
            p = pn;
            if (((r + 1) & 1) == 0) s += coef_[(r + 1) / 2] * p;
        }
        return s;
    }
    std::vector<double> coef_;
    double norm_ = 1.0;
};

}  // namespace imager
