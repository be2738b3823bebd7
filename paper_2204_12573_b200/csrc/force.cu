// force.cu -- steps a6 + a7: back-propagation of dE/dB through A to per-pair forces, and the
// atomics-free force gather ("reordering the summation" so that grad d_i is never formed).
//
// k_backprop, one warp per atom k (row of the current chunk):
//   E_k   = sum of the energy tiles' partial row-dots (fixed order)           (Eq. 1)
//   V_k   = same for the variance tiles                                        (Eq. 2)
//   c_p   = dE_k/dB_p = (2/||B||)(W_p - E_k B^_p),  W = beta B^               (R10, R11)
//   G[nu1,lm] = dE_k/dA[nu1,lm] = sum_{nu2} c_{p(nu1,nu2,l)} (1+delta) A[nu2,lm]
//   f_kj  = dE_k/dr_kj = sum_{n,lm} G[s_j n, lm] grad(g~_n Y_lm)(r_kj)   for every neighbour j
// f_kj is stored once per ordered pair.  k_gather then forms, with the reverse-pair index,
//   F_k = sum_j ( f_kj - f_jk )
// reading each pair force exactly twice and writing each atom's force exactly once.
#include "kernels.cuh"

namespace flare {

constexpr int kBpWarps = 4;

__host__ __device__ inline int bp_warp_doubles(int S, int Nv, int L2, int nmaxp, int ld) {
    // A[Nv][L2|1], c[ld], G^T[S][L2][nmaxp]
    return (Nv * (L2 | 1) + ld + S * L2 * nmaxp + 1) & ~1;  // even: keeps every warp's G^T 16-byte aligned
}

__device__ __forceinline__ void dmma884_f(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}

// g[n] = T_n(x) f_c(r), dg[n] = d g[n]/dr for n < n_max, zero above; fully unrolled so that g/dg stay in registers
template <int NMAXP>
__device__ __forceinline__ void radial_fixed(int n_max, double r, double rc, double (&gv)[NMAXP], double (&dgv)[NMAXP]) {
    const double inv_rc = 1.0 / rc;
    const double q = r * inv_rc;
    const double x = 2.0 * q - 1.0;
    double sn, cs;
    sincospi(q, &sn, &cs);
    const double fc = 0.5 * (1.0 + cs);
    const double dfc = -0.5 * kPi * inv_rc * sn;
    const double dxdr = 2.0 * inv_rc;
    double t0 = 1.0, t1 = x, u0 = 0.0, u1 = 1.0;
#pragma unroll
    for (int n = 0; n < NMAXP; n++) {
        const bool on = n < n_max;
        gv[n] = on ? t0 * fc : 0.0;
        dgv[n] = on ? dxdr * ((double)n * u0) * fc + t0 * dfc : 0.0;
        const double t2 = 2.0 * x * t1 - t0;
        t0 = t1; t1 = t2;
        const double u2 = 2.0 * x * u1 - u0;
        u0 = u1; u1 = u2;
    }
}

template <int LMAX, int NMAXP>
__global__ void __launch_bounds__(kBpWarps * 32)
k_backprop(Grid g, Basis bs, YNorm yn, const AtomS* __restrict__ atoms, const int* __restrict__ nbr_cnt,
           const int* __restrict__ nbr_idx, int mmax, const int* __restrict__ atom_of_row,
           const unsigned char* __restrict__ gid, const GroupDev* __restrict__ groups, int row0, int nrows,
           const double* __restrict__ A_in, const double* __restrict__ Bh, const double* __restrict__ W,
           const double* __restrict__ nrm_in, const double* __restrict__ part, int ld, int chunk_cap, int max_ntn,
           int want_variance, double* __restrict__ pairf, double* __restrict__ e_s, double* __restrict__ v_s) {
    constexpr int L = LMAX + 1;
    constexpr int L2 = L * L;
    constexpr int AS = L2 | 1;
    constexpr int NBL = (2 * LMAX + 1 + 7) / 8;  // n8 blocks needed for the widest m range
    extern __shared__ __align__(16) double smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int local = blockIdx.x * kBpWarps + warp;
    if (local >= nrows) return;
    const int g8 = lane >> 2, t4 = lane & 3;
    const int Nv = bs.Nv;
    double* Gt = smem + (size_t)warp * bp_warp_doubles(bs.S, Nv, L2, NMAXP, ld);  // [S][L2][NMAXP], 16-byte aligned
    double* As = Gt + bs.S * L2 * NMAXP;
    double* cs = As + Nv * AS;

    const int k = atom_of_row[row0 + local];
    const GroupDev gd = groups[gid[k]];

    // ---- E, V from the tile partials (fixed order => deterministic)
    double E = 0.0, V = 0.0;
    for (int t = 0; t < gd.ntn; t++) E += part[(size_t)t * chunk_cap + local];
    if (want_variance)
        for (int t = 0; t < gd.ntn; t++) V += part[((size_t)max_ntn + t) * chunk_cap + local];
    const double nrm = nrm_in[local];
    const double two_inv = (nrm > 0.0) ? 2.0 / nrm : 0.0;
    if (lane == 0) { e_s[k] = E; v_s[k] = V; }
    if (gd.P == 0) return;  // no neighbours (R8): E = V = 0 and no pair forces; the group has no tables

    // ---- stage A, zero G^T, stage c = dE/dB with the diagonal pairs pre-doubled (the 1 + delta factor)
    const double* arow = A_in + (size_t)local * bs.NvL2;
    for (int c = lane; c < bs.NvL2; c += 32) {
        const int nu = c / L2;
        As[nu * AS + (c - nu * L2)] = arow[c];
    }
    for (int c = lane; c < bs.S * L2 * NMAXP; c += 32) Gt[c] = 0.0;
    const double* wrow = W + (size_t)local * ld;
    const double* brow = Bh + (size_t)local * ld;
    for (int p = lane; p < gd.P; p += 32) {
        const int t = __ldg(gd.table + p / L);
        const double dbl = ((t & 255) == (t >> 8)) ? 2.0 : 1.0;
        cs[p] = dbl * two_inv * (wrow[p] - E * brow[p]);
    }
    __syncwarp();

    // ---- G[nu1, (l,m)] = sum_nu2 C_l[nu1,nu2] A[nu2,(l,m)] with C_l[nu1,nu2] = c[q(nu1,nu2) L + l]: per l a small
    // symmetric-matrix product on the tensor pipe.  A-operand (row nu1 = 8mb+g8, col nu2 = k0+t4),
    // B-operand (row nu2 = k0+t4, col m = 8nb+g8), C (row nu1, cols m = 8nb+2t4, +1).
    for (int mb = 0; mb * 8 < Nv; mb++) {
        const int nu1 = mb * 8 + g8;
        double acc[L][NBL][2];
#pragma unroll
        for (int l = 0; l < L; l++)
#pragma unroll
            for (int nb = 0; nb < NBL; nb++) { acc[l][nb][0] = 0.0; acc[l][nb][1] = 0.0; }
        for (int k0 = 0; k0 < Nv; k0 += 4) {
            const int nu2 = k0 + t4;
            const bool in = nu1 < Nv && nu2 < Nv;
            const int q = in ? __ldg(gd.lut + nu1 * Nv + nu2) : -1;
            const double* a2 = As + (nu2 < Nv ? nu2 : 0) * AS;
#pragma unroll
            for (int l = 0; l < L; l++) {
                const double a = (q >= 0) ? cs[q * L + l] : 0.0;
#pragma unroll
                for (int nb = 0; nb < NBL; nb++) {
                    if (nb * 8 < 2 * l + 1) {
                        const int m = nb * 8 + g8;
                        const double b = (nu2 < Nv && m < 2 * l + 1) ? a2[l * l + m] : 0.0;
                        dmma884_f(acc[l][nb][0], acc[l][nb][1], a, b);
                    }
                }
            }
        }
        if (nu1 < Nv) {
            const int s1 = nu1 / bs.n_max, n1 = nu1 - s1 * bs.n_max;
            double* gt = Gt + (size_t)s1 * L2 * NMAXP + n1;
#pragma unroll
            for (int l = 0; l < L; l++)
#pragma unroll
                for (int nb = 0; nb < NBL; nb++) {
                    const int m = nb * 8 + 2 * t4;
                    if (m < 2 * l + 1) gt[(l * l + m) * NMAXP] = acc[l][nb][0];
                    if (m + 1 < 2 * l + 1) gt[(l * l + m + 1) * NMAXP] = acc[l][nb][1];
                }
        }
    }
    __syncwarp();

    // ---- per-pair forces f_kj = sum_{n,lm} G[s_j n, lm] grad(g~_n Y_lm)(r_kj): lanes over neighbours
    const AtomS me = load_atom(atoms + k);
    const int cnt = nbr_cnt[k];
    for (int base = 0; base < cnt; base += 32) {
        const int s = base + lane;
        if (s < cnt) {
            const int j = nbr_idx[(size_t)k * mmax + s];
            const AtomS o = load_atom(atoms + j);
            double dx, dy, dz;
            displacement(g, me, o, dx, dy, dz);
            const double r = sqrt(dx * dx + dy * dy + dz * dz);
            const double ir = 1.0 / r;
            const double ux = dx * ir, uy = dy * ir, uz = dz * ir;
            double gr[NMAXP], dgr[NMAXP];
            radial_fixed<NMAXP>(bs.n_max, r, bs.rc[me.type * bs.S + o.type], gr, dgr);
            const double* Gj = Gt + (size_t)o.type * L2 * NMAXP;
            double srad = 0.0, vx = 0.0, vy = 0.0, vz = 0.0;
            real_ylm<LMAX, true>(yn, ux, uy, uz, [&](int lm, double Y, double gx, double gy, double gz) {
                const double2* gp = reinterpret_cast<const double2*>(Gj + lm * NMAXP);
                double hr = 0.0, hg = 0.0;  // sum_n G[n,lm] dg_n  and  sum_n G[n,lm] g_n
#pragma unroll
                for (int n2 = 0; n2 < NMAXP / 2; n2++) {
                    const double2 Gv = gp[n2];
                    hr = fma(Gv.x, dgr[2 * n2], hr);
                    hr = fma(Gv.y, dgr[2 * n2 + 1], hr);
                    hg = fma(Gv.x, gr[2 * n2], hg);
                    hg = fma(Gv.y, gr[2 * n2 + 1], hg);
                }
                srad = fma(hr, Y, srad);
                vx = fma(hg, gx, vx);
                vy = fma(hg, gy, vy);
                vz = fma(hg, gz, vz);
            });
            // grad Y = (1/r)(I - u u^T) grad_u Y~ ; radial part along u
            const double udv = ux * vx + uy * vy + uz * vz;
            double* pf = pairf + ((size_t)k * mmax + s) * 3;
            pf[0] = srad * ux + (vx - ux * udv) * ir;
            pf[1] = srad * uy + (vy - uy * udv) * ir;
            pf[2] = srad * uz + (vz - uz * udv) * ir;
        }
    }
}

template <int LMAX, int NMAXP>
static void launch_backprop(Launcher& L, const Grid& g, const Basis& bs, const YNorm& yn, const Workspace& ws,
                            int mmax, const GroupDev* groups, int row0, int nrows, int ld, int chunk_cap, int max_ntn,
                            bool want_variance) {
    constexpr int L2 = (LMAX + 1) * (LMAX + 1);
    const size_t smem = sizeof(double) * kBpWarps * (size_t)bp_warp_doubles(bs.S, bs.Nv, L2, NMAXP, ld);
    static size_t configured = 0;
    if (smem > 48 * 1024 && smem > configured) {
        cudaFuncSetAttribute(k_backprop<LMAX, NMAXP>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        configured = smem;
    }
    L.launch(k_backprop<LMAX, NMAXP>, dim3((nrows + kBpWarps - 1) / kBpWarps), dim3(kBpWarps * 32), smem, g, bs, yn,
             (const AtomS*)ws.atoms, (const int*)ws.nbr_cnt, (const int*)ws.nbr_idx, mmax,
             (const int*)ws.atom_of_row, (const unsigned char*)ws.gid, groups, row0, nrows, (const double*)ws.A,
             (const double*)ws.Bh, (const double*)ws.W, (const double*)ws.nrm, (const double*)ws.part, ld, chunk_cap,
             max_ntn, want_variance ? 1 : 0, ws.pairf, ws.e_s, ws.v_s);
}

void run_backprop(Launcher& L, const Grid& g, const Basis& bs, const YNorm& yn, const Workspace& ws, int mmax,
                  const GroupDev* groups, int row0, int nrows, int ld, int chunk_cap, int max_ntn,
                  bool want_variance) {
    if (nrows <= 0) return;
#define FLARE_CASE(LM)                                                                                                \
    case LM:                                                                                                          \
        if (bs.n_max <= 8)                                                                                            \
            launch_backprop<LM, 8>(L, g, bs, yn, ws, mmax, groups, row0, nrows, ld, chunk_cap, max_ntn, want_variance); \
        else                                                                                                          \
            launch_backprop<LM, 16>(L, g, bs, yn, ws, mmax, groups, row0, nrows, ld, chunk_cap, max_ntn, want_variance); \
        break;
    switch (bs.l_max) {
        FLARE_CASE(0) FLARE_CASE(1) FLARE_CASE(2) FLARE_CASE(3) FLARE_CASE(4) FLARE_CASE(5) FLARE_CASE(6)
        default: break;
    }
#undef FLARE_CASE
}

// ------------------------------------------------------------------ a7: atomics-free gather
constexpr int kGatherWarps = 8;

__global__ void __launch_bounds__(kGatherWarps * 32)
k_gather(int n, int mmax, const AtomS* __restrict__ atoms, const int* __restrict__ nbr_cnt,
         const int* __restrict__ nbr_idx, const unsigned char* __restrict__ rev, const double* __restrict__ pairf,
         const double* __restrict__ e_s, const double* __restrict__ v_s, double* __restrict__ e_out,
         double* __restrict__ f_out, double* __restrict__ var_out) {
    const int lane = threadIdx.x & 31;
    const int k = blockIdx.x * kGatherWarps + (threadIdx.x >> 5);
    if (k >= n) return;
    const int cnt = nbr_cnt[k];
    double fx = 0.0, fy = 0.0, fz = 0.0;
    for (int s = lane; s < cnt; s += 32) {
        const size_t own = ((size_t)k * mmax + s) * 3;
        const int j = nbr_idx[(size_t)k * mmax + s];
        const size_t oth = ((size_t)j * mmax + rev[(size_t)k * mmax + s]) * 3;
        fx += pairf[own] - pairf[oth];
        fy += pairf[own + 1] - pairf[oth + 1];
        fz += pairf[own + 2] - pairf[oth + 2];
    }
    fx = warp_sum(fx); fy = warp_sum(fy); fz = warp_sum(fz);
    if (lane == 0) {
        const int i = atoms[k].orig;
        if (f_out) { f_out[3 * (size_t)i] = fx; f_out[3 * (size_t)i + 1] = fy; f_out[3 * (size_t)i + 2] = fz; }
        if (e_out) e_out[i] = e_s[k];
        if (var_out) var_out[i] = v_s[k];
    }
}

void run_gather(Launcher& L, const Workspace& ws, int n, int mmax, double* e_out, double* f_out, double* var_out) {
    if (n <= 0) return;
    L.launch(k_gather, dim3((n + kGatherWarps - 1) / kGatherWarps), dim3(kGatherWarps * 32), 0, n, mmax,
             (const AtomS*)ws.atoms, (const int*)ws.nbr_cnt, (const int*)ws.nbr_idx, (const unsigned char*)ws.rev,
             (const double*)ws.pairf, (const double*)ws.e_s, (const double*)ws.v_s, e_out, f_out, var_out);
}

}  // namespace flare
