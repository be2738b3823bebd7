// integrate.cu -- step a9: velocity-Verlet NVE (BASELINE.json north_star; R12, R13).
//   kick+drift:  v += (dt/2) kappa F/m ;  x += dt v ;  x wrapped into the box (canonical wrap, R6)
//   kick:        v += (dt/2) kappa F/m
// Pure streaming kernels over 3N doubles (HBM-bound: 120 B/atom fused).
#include "kernels.cuh"

namespace flare {

__global__ void k_kick_drift(Grid g, int n, double* __restrict__ x, double* __restrict__ v,
                             const double* __restrict__ f, const int* __restrict__ types,
                             const double* __restrict__ accel_half_dt, double dt) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int t = types[i];
    const double a = (unsigned)t < (unsigned)kMaxSpecies ? accel_half_dt[t] : 0.0;  // a bad type is flagged by the evaluation
#pragma unroll
    for (int d = 0; d < 3; d++) {
        const size_t q = 3 * (size_t)i + d;
        const double vn = v[q] + a * f[q];
        double xn = x[q] + dt * vn;
        if (g.pbc[d]) xn = wrap_coord(xn, g.L[d]);
        v[q] = vn;
        x[q] = xn;
    }
}

__global__ void k_kick(int n, double* __restrict__ v, const double* __restrict__ f, const int* __restrict__ types,
                       const double* __restrict__ accel_half_dt) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int t = types[i];
    const double a = (unsigned)t < (unsigned)kMaxSpecies ? accel_half_dt[t] : 0.0;  // a bad type is flagged by the evaluation
#pragma unroll
    for (int d = 0; d < 3; d++) {
        const size_t q = 3 * (size_t)i + d;
        v[q] += a * f[q];
    }
}

void run_kick_drift(Launcher& L, const Grid& g, int n, double* x, double* v, const double* f, const int* types,
                    const double* accel_half_dt, double dt) {
    if (n <= 0) return;
    L.launch(k_kick_drift, dim3((n + 255) / 256), dim3(256), 0, g, n, x, v, f, types, accel_half_dt, dt);
}

void run_kick(Launcher& L, int n, double* v, const double* f, const int* types, const double* accel_half_dt) {
    if (n <= 0) return;
    L.launch(k_kick, dim3((n + 255) / 256), dim3(256), 0, n, v, f, types, accel_half_dt);
}

}  // namespace flare
