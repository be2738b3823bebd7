// basis.cuh -- per-pair basis of the ACE-B2 descriptor ("spherical harmonics and radial
// functions"; readings R1-R3): Chebyshev T_n(2r/r_c - 1) times the cosine cutoff, and
// real orthonormal Y_lm evaluated without any division by sin(theta).
#pragma once
#include "common.cuh"

namespace flare {

// K_lm sqrt(2 - delta_m0), K_lm = sqrt((2l+1)/(4 pi) (l-m)!/(l+m)!), index l(l+1)/2 + m.
struct YNorm {
    double k[(kMaxLmax + 1) * (kMaxLmax + 2) / 2];
};

constexpr double kPi = 3.14159265358979323846;

__host__ __device__ constexpr double double_factorial_odd(int m) {  // (2m-1)!!
    double f = 1.0;
    for (int i = 1; i <= m; i++) f *= (double)(2 * i - 1);
    return f;
}

// Radial functions of one pair: g[n] = T_n(x) f_c(r), and (GRAD) dg[n] = d g[n] / dr,
//   x = 2r/r_c - 1, f_c = (1 + cos(pi r/r_c))/2, T_n' = n U_{n-1}.
// `put(n, g, dg)` consumes each value (so callers choose registers or shared memory).
template <bool GRAD, class Put>
__device__ __forceinline__ void radial_basis(int n_max, double r, double rc, Put&& put) {
    const double inv_rc = 1.0 / rc;
    const double q = r * inv_rc;
    const double x = 2.0 * q - 1.0;
    double sn, cs;
    sincospi(q, &sn, &cs);
    const double fc = 0.5 * (1.0 + cs);
    const double dfc = -0.5 * kPi * inv_rc * sn;
    const double dxdr = 2.0 * inv_rc;
    double t0 = 1.0, t1 = x;    // T_{n}, T_{n+1}
    double u0 = 0.0, u1 = 1.0;  // U_{n-1}, U_{n}   (U_{-1} = 0, U_0 = 1)
    for (int n = 0; n < n_max; n++) {
        double dg = 0.0;
        if (GRAD) dg = dxdr * ((double)n * u0) * fc + t0 * dfc;
        put(n, t0 * fc, dg);
        double t2 = 2.0 * x * t1 - t0;
        t0 = t1; t1 = t2;
        double u2 = 2.0 * x * u1 - u0;
        u0 = u1; u1 = u2;
    }
}

// Real spherical harmonics of a unit vector (x,y,z), l <= LMAX, index lm = l*l + l + m:
//   Y_l0 = K Q_l^0(z);  Y_l,+m = K Q_l^m(z) C_m;  Y_l,-m = K Q_l^m(z) S_m;  C_m + i S_m = (x+iy)^m,
// with Q_l^m(z) = P_l^m(z) / (1-z^2)^{m/2} from the three-term recurrence in l at fixed m:
//   Q_m^m = (2m-1)!!,  Q_{m+1}^m = (2m+1) z Q_m^m,  (l-m) Q_l^m = (2l-1) z Q_{l-1}^m - (l+m-1) Q_{l-2}^m,
// and dQ_l^m/dz = Q_l^{m+1} (carried alongside).  With GRAD, (gx,gy,gz) is the gradient of the
// polynomial extension K Q_l^m(z) C_m(x,y) with respect to (x,y,z); callers project it onto the
// tangent plane: grad Y_lm = (1/r)(I - u u^T) (gx,gy,gz).
// `emit(lm, Y, gx, gy, gz)` is called once per (l,m); lm is a compile-time constant after unrolling.
template <int LMAX, bool GRAD, class Emit>
__device__ __forceinline__ void real_ylm(const YNorm& yn, double x, double y, double z, Emit&& emit) {
    double cm = 1.0, sm = 0.0;    // C_m, S_m
    double cm1 = 0.0, sm1 = 0.0;  // C_{m-1}, S_{m-1}
#pragma unroll
    for (int m = 0; m <= LMAX; m++) {
        // recurrences in l for Q^m (qa) and Q^{m+1} (qb)
        double qa = double_factorial_odd(m), qa1 = 0.0;  // Q_l^m, Q_{l-1}^m at l = m
        double qb = 0.0, qb1 = 0.0;                      // Q_l^{m+1}, Q_{l-1}^{m+1} at l = m  (zero: l < m+1)
#pragma unroll
        for (int l = m; l <= LMAX; l++) {
            const double K = yn.k[l * (l + 1) / 2 + m];
            const double kq = K * qa;
            if (m == 0) {
                emit(l * l + l, kq, 0.0, 0.0, GRAD ? K * qb : 0.0);
            } else {
                const double dm = (double)m;
                emit(l * l + l + m, kq * cm, GRAD ? kq * dm * cm1 : 0.0, GRAD ? -kq * dm * sm1 : 0.0,
                     GRAD ? K * qb * cm : 0.0);
                emit(l * l + l - m, kq * sm, GRAD ? kq * dm * sm1 : 0.0, GRAD ? kq * dm * cm1 : 0.0,
                     GRAD ? K * qb * sm : 0.0);
            }
            if (l < LMAX) {
                // advance l -> l+1
                const int l1 = l + 1;
                double qn = ((2.0 * l1 - 1.0) * z * qa - (double)(l1 + m - 1) * qa1) * (1.0 / (double)(l1 - m));
                qa1 = qa; qa = qn;
                if (GRAD) {
                    double bn;
                    if (l1 == m + 1) bn = double_factorial_odd(m + 1);
                    else bn = ((2.0 * l1 - 1.0) * z * qb - (double)(l1 + m) * qb1) * (1.0 / (double)(l1 - m - 1));
                    qb1 = qb; qb = bn;
                }
            }
        }
        // (x+iy)^{m+1}
        const double cn = x * cm - y * sm;
        const double sn = x * sm + y * cm;
        cm1 = cm; sm1 = sm;
        cm = cn; sm = sn;
    }
}

}  // namespace flare
