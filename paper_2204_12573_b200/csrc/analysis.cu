// analysis.cu -- SURVEY.md 8(f) rows #2 and #3, from quantities the force evaluation already holds:
//   * the virial Xi_ab = dE/d eps_ab = sum_i sum_{j in N(i)} (dE_i/dr_ij)_a (r_ij)_b  (stress),
//     a reduction over the stored per-pair forces;
//   * the on-the-fly analysis of the paper's production run: maximum uncertainty sqrt(V_i) and the number of
//     atoms above a threshold, coordination numbers from the neighbour list ("another H
//     within 1 A");
//   * the half steps of a Nose-Hoover thermostat (R19).
// All reductions are two-stage with a fixed assignment of atoms to blocks and a fixed summation order, so
// results are bit-reproducible run to run; integer counts and the maximum use atomics (order-independent).
#include "kernels.cuh"

namespace flare {

constexpr int kRedBlocks = 1184;  // 148 SMs x 8
constexpr int kRedThreads = 256;

// sum v over the block in a fixed order; result valid in thread 0
template <int NV>
__device__ __forceinline__ void block_sum(double (&v)[NV], double* sm /*[8][NV]*/) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
    for (int q = 0; q < NV; q++) v[q] = warp_sum(v[q]);
    if (lane == 0)
#pragma unroll
        for (int q = 0; q < NV; q++) sm[w * NV + q] = v[q];
    __syncthreads();
    if (threadIdx.x == 0)
#pragma unroll
        for (int q = 0; q < NV; q++) {
            double t = 0.0;
            for (int ww = 0; ww < kRedThreads / 32; ww++) t += sm[ww * NV + q];
            v[q] = t;
        }
}

// final stage: one block sums the per-block partials [n_part][NV] in a fixed order
template <int NV>
__global__ void __launch_bounds__(kRedThreads) k_reduce_final(int n_part, const double* __restrict__ part,
                                                               double* __restrict__ out) {
    __shared__ double sm[(kRedThreads / 32) * NV];
    double v[NV];
#pragma unroll
    for (int q = 0; q < NV; q++) v[q] = 0.0;
    for (int b = threadIdx.x; b < n_part; b += kRedThreads)
#pragma unroll
        for (int q = 0; q < NV; q++) v[q] += part[(size_t)b * NV + q];
    block_sum<NV>(v, sm);
    if (threadIdx.x == 0)
#pragma unroll
        for (int q = 0; q < NV; q++) out[q] = v[q];
}

// ------------------------------------------------------------------ virial
__global__ void __launch_bounds__(kRedThreads)
k_virial_partial(Grid g, int n, int mmax, const AtomS* __restrict__ atoms, const int* __restrict__ nbr_cnt,
                 const int* __restrict__ nbr_idx, const double* __restrict__ pairf, double* __restrict__ part) {
    __shared__ double sm[(kRedThreads / 32) * 9];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    double v[9];
#pragma unroll
    for (int q = 0; q < 9; q++) v[q] = 0.0;
    // warp per atom, atoms dealt to (block, warp) in a fixed pattern
    for (int k = blockIdx.x * (kRedThreads / 32) + w; k < n; k += gridDim.x * (kRedThreads / 32)) {
        const AtomS me = load_atom(atoms + k);
        const int cnt = nbr_cnt[k];
        for (int s = lane; s < cnt; s += 32) {
            const AtomS o = load_atom(atoms + nbr_idx[(size_t)k * mmax + s]);
            double d[3];
            displacement(g, me, o, d[0], d[1], d[2]);
            const double* pf = pairf + ((size_t)k * mmax + s) * 3;
#pragma unroll
            for (int a = 0; a < 3; a++)
#pragma unroll
                for (int b = 0; b < 3; b++) v[3 * a + b] = fma(pf[a], d[b], v[3 * a + b]);
        }
    }
    block_sum<9>(v, sm);
    if (threadIdx.x == 0)
#pragma unroll
        for (int q = 0; q < 9; q++) part[(size_t)blockIdx.x * 9 + q] = v[q];
}

void run_virial(Launcher& L, const Grid& g, const Workspace& ws, int n, int mmax, double* out9) {
    L.launch(k_virial_partial, dim3(kRedBlocks), dim3(kRedThreads), 0, g, n, mmax, (const AtomS*)ws.atoms,
             (const int*)ws.nbr_cnt, (const int*)ws.nbr_idx, (const double*)ws.pairf, ws.red);
    L.launch(k_reduce_final<9>, dim3(1), dim3(kRedThreads), 0, kRedBlocks, (const double*)ws.red, out9);
}

// ------------------------------------------------------------------ uncertainty + coordination analysis
// out: [0] max sqrt(max(V,0)) as the bits of a non-negative double, [1] count above threshold, [2..17] histogram
// of the coordination numbers of species_a atoms (last bin: >= 15).  coord (caller's atom order) may be null.
__global__ void __launch_bounds__(kRedThreads)
k_analyze(Grid g, int n, int mmax, const AtomS* __restrict__ atoms, const int* __restrict__ nbr_cnt,
          const int* __restrict__ nbr_idx, const double* __restrict__ v_s, int have_var, double threshold,
          int species_a, int species_b, double r_coord2, int want_coord, int* __restrict__ coord,
          unsigned long long* __restrict__ out) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    double u = 0.0;
    int above = 0;
    if (k < n && have_var) {
        const double V = v_s[k];
        u = sqrt(V > 0.0 ? V : 0.0);
        above = u > threshold ? 1 : 0;
    }
    if (have_var) {
        // non-negative doubles order like their bit patterns
        unsigned long long bits = (unsigned long long)__double_as_longlong(u);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const unsigned long long t = __shfl_xor_sync(kFull, bits, o);
            bits = t > bits ? t : bits;
        }
        const unsigned m = __ballot_sync(kFull, above);
        if ((threadIdx.x & 31) == 0) {
            atomicMax(out, bits);
            if (m) atomicAdd(out + 1, (unsigned long long)__popc(m));
        }
    }
    if (k < n && want_coord) {
        const AtomS me = load_atom(atoms + k);
        int c = 0;
        if (me.type == species_a) {
            const int cnt = nbr_cnt[k];
            for (int s = 0; s < cnt; s++) {
                const AtomS o = load_atom(atoms + nbr_idx[(size_t)k * mmax + s]);
                if (o.type != species_b) continue;
                double dx, dy, dz;
                displacement(g, me, o, dx, dy, dz);
                if (dist2_canonical(dx, dy, dz) < r_coord2) c++;  // same canonical arithmetic as the neighbour test (R6)
            }
            atomicAdd(out + 2 + min(c, 15), 1ull);
        }
        if (coord) coord[me.orig] = c;
    }
}

void run_analyze(Launcher& L, const Grid& g, const Workspace& ws, int n, int mmax, bool have_var, double threshold,
                 int species_a, int species_b, double r_coord, bool want_coord, int* coord,
                 unsigned long long* out18) {
    L.memset(out18, 0, sizeof(unsigned long long) * 18);
    L.launch(k_analyze, dim3((n + kRedThreads - 1) / kRedThreads), dim3(kRedThreads), 0, g, n, mmax,
             (const AtomS*)ws.atoms, (const int*)ws.nbr_cnt, (const int*)ws.nbr_idx, (const double*)ws.v_s,
             have_var ? 1 : 0, threshold, species_a, species_b, r_coord * r_coord, want_coord ? 1 : 0, coord, out18);
}

// ------------------------------------------------------------------ Nose-Hoover half step (R19)
//   K2 = sum m v^2 / kappa;  xi += (h/2)(K2 - g kT)/Q;  s = exp(-xi h);  v *= s;  K2 *= s^2;  eta += xi h;
//   xi += (h/2)(K2 - g kT)/Q
// thermo (device): [0] xi, [1] eta, [2] scale s, [3] K2 before the half step (diagnostic)
__global__ void __launch_bounds__(kRedThreads)
k_ke_partial(int n, const double* __restrict__ v, const int* __restrict__ types, const double* __restrict__ mass,
             double inv_kappa, double* __restrict__ part) {
    __shared__ double sm[kRedThreads / 32];
    double t[1] = {0.0};
    for (int i = blockIdx.x * kRedThreads + threadIdx.x; i < n; i += gridDim.x * kRedThreads) {
        const int ty = types[i];
        const double m = (unsigned)ty < (unsigned)kMaxSpecies ? mass[ty] : 0.0;
        const double vx = v[3 * (size_t)i], vy = v[3 * (size_t)i + 1], vz = v[3 * (size_t)i + 2];
        t[0] += m * (vx * vx + vy * vy + vz * vz) * inv_kappa;
    }
    block_sum<1>(t, sm);
    if (threadIdx.x == 0) part[blockIdx.x] = t[0];
}

__global__ void __launch_bounds__(kRedThreads)
k_nh_update(int n_part, const double* __restrict__ part, double h, double gkT, double Q, double* __restrict__ thermo) {
    __shared__ double sm[kRedThreads / 32];
    double t[1] = {0.0};
    for (int b = threadIdx.x; b < n_part; b += kRedThreads) t[0] += part[b];
    block_sum<1>(t, sm);
    if (threadIdx.x == 0) {
        double K2 = t[0];
        double xi = thermo[0], eta = thermo[1];
        thermo[3] = K2;
        xi += 0.5 * h * (K2 - gkT) / Q;
        const double s = exp(-xi * h);
        K2 *= s * s;
        eta += xi * h;
        xi += 0.5 * h * (K2 - gkT) / Q;
        thermo[0] = xi; thermo[1] = eta; thermo[2] = s;
    }
}

__global__ void k_scale_v(size_t n3, double* __restrict__ v, const double* __restrict__ thermo) {
    const size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
    if (i < n3) v[i] *= thermo[2];
}

void run_nh_half(Launcher& L, const Workspace& ws, int n, const double* mass_dev, double h, double gkT, double Q,
                 double* thermo) {
    if (n <= 0) return;
    L.launch(k_ke_partial, dim3(kRedBlocks), dim3(kRedThreads), 0, n, (const double*)ws.v, (const int*)ws.types, mass_dev,
             1.0 / 9.648533212331e-3, ws.red);
    L.launch(k_nh_update, dim3(1), dim3(kRedThreads), 0, kRedBlocks, (const double*)ws.red, h, gkT, Q, thermo);
    const size_t n3 = 3 * (size_t)n;
    L.launch(k_scale_v, dim3((unsigned)((n3 + 255) / 256)), dim3(256), 0, n3, ws.v, (const double*)thermo);
}

}  // namespace flare
