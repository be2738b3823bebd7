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

__host__ __device__ inline int bp_warp_doubles(int n_max, int NvL2, int ld) {
    // A, G : NvL2 each; c : ld; per-lane radial values g, dg : 2 * n_max * 32
    return 2 * NvL2 + ld + 2 * n_max * 32;
}

template <int LMAX>
__global__ void __launch_bounds__(kBpWarps * 32)
k_backprop(Grid g, Basis bs, YNorm yn, const AtomS* __restrict__ atoms, const int* __restrict__ nbr_cnt,
           const int* __restrict__ nbr_idx, int mmax, const int* __restrict__ atom_of_row,
           const unsigned char* __restrict__ gid, const GroupDev* __restrict__ groups, int row0, int nrows,
           const double* __restrict__ A_in, const double* __restrict__ Bh, const double* __restrict__ W,
           const double* __restrict__ nrm_in, const double* __restrict__ part, int ld, int chunk_cap, int max_ntn,
           int want_variance, double* __restrict__ pairf, double* __restrict__ e_s, double* __restrict__ v_s) {
    constexpr int L2 = (LMAX + 1) * (LMAX + 1);
    extern __shared__ double smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int local = blockIdx.x * kBpWarps + warp;
    if (local >= nrows) return;
    double* As = smem + (size_t)warp * bp_warp_doubles(bs.n_max, bs.NvL2, ld);
    double* Gs = As + bs.NvL2;
    double* cs = Gs + bs.NvL2;
    double* gl = cs + ld;                 // [n_max][32] this lane's g~_n
    double* dgl = gl + bs.n_max * 32;     // [n_max][32] this lane's d g~_n / dr

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

    // ---- stage A and c = dE/dB
    const double* arow = A_in + (size_t)local * bs.NvL2;
    for (int c = lane; c < bs.NvL2; c += 32) { As[c] = arow[c]; Gs[c] = 0.0; }
    const double* wrow = W + (size_t)local * ld;
    const double* brow = Bh + (size_t)local * ld;
    for (int p = lane; p < gd.P; p += 32) cs[p] = two_inv * (wrow[p] - E * brow[p]);
    __syncwarp();

    // ---- G[nu1,lm] = sum_nu2 c_p (1+delta) A[nu2,lm]: lanes own (nu1,lm); loop the group's components.
    // The component table is ordered (nu1, nu2>=nu1, l), so for a fixed (nu, l) the components with
    // nu as FIRST index are contiguous in nu2 and those with nu as SECOND index are found by table walk;
    // with P up to a few thousand a direct walk over p per lane would be wasteful, so each lane walks
    // only the (nu2) partners of its own (nu1, l) through the closed-form index of the dense ordering
    // when the group is dense, and through the table otherwise.
    {
        const int Nv = bs.Nv;
        const int L = LMAX + 1;
        for (int c = lane; c < bs.NvL2; c += 32) {
            const int v1 = c / L2, lm = c - v1 * L2;
            int l = 0;
            while ((l + 1) * (l + 1) <= lm) l++;
            double acc = 0.0;
            if (gd.P == bs.P) {
                // dense ordering: p(a<=b, l) = (a*Nv - a(a-1)/2 + (b-a))*L + l
                for (int v2 = 0; v2 < Nv; v2++) {
                    const int a = min(v1, v2), b = max(v1, v2);
                    const int p = (a * Nv - (a * (a - 1)) / 2 + (b - a)) * L + l;
                    const double w = (v1 == v2) ? 2.0 : 1.0;
                    acc = fma(w * cs[p], As[v2 * L2 + lm], acc);
                }
            } else {
                for (int p = 0; p < gd.P; p++) {
                    const int t = __ldg(gd.table + p);
                    const int a = t & 255, b = (t >> 8) & 255, ll = t >> 16;
                    if (ll != l) continue;
                    if (a == v1) acc = fma((a == b ? 2.0 : 1.0) * cs[p], As[b * L2 + lm], acc);
                    else if (b == v1) acc = fma(cs[p], As[a * L2 + lm], acc);
                }
            }
            Gs[c] = acc;
        }
    }
    __syncwarp();

    // ---- per-pair forces: lanes over neighbours
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
            radial_basis<true>(bs.n_max, r, bs.rc[me.type * bs.S + o.type],
                               [&](int n, double gv, double dgv) { gl[n * 32 + lane] = gv; dgl[n * 32 + lane] = dgv; });
            const double* Gj = Gs + o.type * bs.n_max * L2;
            double srad = 0.0, vx = 0.0, vy = 0.0, vz = 0.0;
            real_ylm<LMAX, true>(yn, ux, uy, uz, [&](int lm, double Y, double gx, double gy, double gz) {
                double hr = 0.0, hg = 0.0;  // sum_n G[n,lm] dg_n  and  sum_n G[n,lm] g_n
                for (int n = 0; n < bs.n_max; n++) {
                    const double Gv = Gj[n * L2 + lm];
                    hr = fma(Gv, dgl[n * 32 + lane], hr);
                    hg = fma(Gv, gl[n * 32 + lane], hg);
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

template <int LMAX>
static void launch_backprop(Launcher& L, const Grid& g, const Basis& bs, const YNorm& yn, const Workspace& ws,
                            int mmax, const GroupDev* groups, int row0, int nrows, int ld, int chunk_cap, int max_ntn,
                            bool want_variance) {
    const size_t smem = sizeof(double) * kBpWarps * (size_t)bp_warp_doubles(bs.n_max, bs.NvL2, ld);
    static size_t configured = 0;
    if (smem > 48 * 1024 && smem > configured) {
        cudaFuncSetAttribute(k_backprop<LMAX>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        configured = smem;
    }
    L.launch(k_backprop<LMAX>, dim3((nrows + kBpWarps - 1) / kBpWarps), dim3(kBpWarps * 32), smem, g, bs, yn,
             (const AtomS*)ws.atoms, (const int*)ws.nbr_cnt, (const int*)ws.nbr_idx, mmax,
             (const int*)ws.atom_of_row, (const unsigned char*)ws.gid, groups, row0, nrows, (const double*)ws.A,
             (const double*)ws.Bh, (const double*)ws.W, (const double*)ws.nrm, (const double*)ws.part, ld, chunk_cap,
             max_ntn, want_variance ? 1 : 0, ws.pairf, ws.e_s, ws.v_s);
}

void run_backprop(Launcher& L, const Grid& g, const Basis& bs, const YNorm& yn, const Workspace& ws, int mmax,
                  const GroupDev* groups, int row0, int nrows, int ld, int chunk_cap, int max_ntn,
                  bool want_variance) {
    if (nrows <= 0) return;
    switch (bs.l_max) {
#define FLARE_CASE(LM) \
    case LM: launch_backprop<LM>(L, g, bs, yn, ws, mmax, groups, row0, nrows, ld, chunk_cap, max_ntn, want_variance); break;
        FLARE_CASE(0) FLARE_CASE(1) FLARE_CASE(2) FLARE_CASE(3) FLARE_CASE(4) FLARE_CASE(5) FLARE_CASE(6)
#undef FLARE_CASE
        default: break;
    }
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
