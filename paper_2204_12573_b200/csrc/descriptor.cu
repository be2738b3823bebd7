// descriptor.cu -- steps a2 + a3: per-pair basis, A accumulation, B2 contraction, normalisation
// (P:L123-129).  One warp per atom: neighbours are spread across lanes for the basis evaluation
// (sqrt, sincospi, Chebyshev and Y_lm recurrences), their g~_n and Y_lm values are staged in shared
// memory, then the lanes switch to owning (n,l,m) components and sum over the staged neighbours
// -- no shuffle reduction over 256+ components is needed.  A stays in shared memory for the B2
// contraction; B^ goes to the quadratic-form row of the atom.
#include "kernels.cuh"

namespace flare {

constexpr int kDescWarps = 4;

__host__ __device__ inline int desc_warp_doubles(int n_max, int L2, int NvL2) {
    return 32 * (n_max | 1) + 32 * (L2 | 1) + NvL2 + 16;
}

template <int LMAX>
__global__ void __launch_bounds__(kDescWarps * 32)
k_descriptor(Grid g, Basis bs, YNorm yn, const AtomS* __restrict__ atoms, const int* __restrict__ nbr_cnt,
             const int* __restrict__ nbr_idx, int mmax, const int* __restrict__ atom_of_row,
             const unsigned char* __restrict__ gid, const GroupDev* __restrict__ groups, int row0, int nrows,
             double* __restrict__ A_out, double* __restrict__ bh_out, int ld, double* __restrict__ nrm_out,
             const int* __restrict__ out_map) {
    constexpr int L2 = (LMAX + 1) * (LMAX + 1);
    constexpr int YS = L2 | 1;
    extern __shared__ double smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int local = blockIdx.x * kDescWarps + warp;
    if (local >= nrows) return;  // warps are independent: only __syncwarp below
    const int GS = bs.n_max | 1;
    const int nL2 = bs.n_max * L2;
    double* gs = smem + (size_t)warp * desc_warp_doubles(bs.n_max, L2, bs.NvL2);
    double* ys = gs + 32 * GS;
    double* As = ys + 32 * YS;
    int* sjs = reinterpret_cast<int*>(As + bs.NvL2);

    const int k = atom_of_row[row0 + local];
    const AtomS me = load_atom(atoms + k);
    const int cnt = nbr_cnt[k];
    for (int c = lane; c < bs.NvL2; c += 32) As[c] = 0.0;

    for (int base = 0; base < cnt; base += 32) {
        const int nact = min(32, cnt - base);
        int sj = -1;
        if (lane < nact) {
            const int j = nbr_idx[(size_t)k * mmax + base + lane];
            const AtomS o = load_atom(atoms + j);
            double dx, dy, dz;
            displacement(g, me, o, dx, dy, dz);
            const double r = sqrt(dx * dx + dy * dy + dz * dz);
            const double ir = 1.0 / r;
            sj = o.type;
            double* gl = gs + lane * GS;
            radial_basis<false>(bs.n_max, r, bs.rc[me.type * bs.S + sj], [&](int n, double gv, double) { gl[n] = gv; });
            double* yl = ys + lane * YS;
            real_ylm<LMAX, false>(yn, dx * ir, dy * ir, dz * ir,
                                  [&](int lm, double Y, double, double, double) { yl[lm] = Y; });
        }
        sjs[lane] = sj;
        __syncwarp();
        for (int s = 0; s < bs.S; s++) {
            if (!__any_sync(kFull, sj == s)) continue;
            for (int c = lane; c < nL2; c += 32) {
                const int n = c / L2, lm = c - n * L2;
                double acc = 0.0;
                for (int jj = 0; jj < nact; jj++)
                    if (sjs[jj] == s) acc = fma(gs[jj * GS + n], ys[jj * YS + lm], acc);
                As[s * nL2 + c] += acc;
            }
        }
        __syncwarp();
    }

    if (A_out) {
        double* arow = A_out + (size_t)local * bs.NvL2;
        for (int c = lane; c < bs.NvL2; c += 32) arow[c] = As[c];
    }

    // B2 contraction: B[nu1<=nu2, l] = sum_m A[nu1,l,m] A[nu2,l,m]; first pass for ||B||, second writes B^
    const GroupDev gd = groups[gid[k]];
    double n2 = 0.0;
    for (int p = lane; p < gd.P; p += 32) {
        const int t = __ldg(gd.table + p);
        const int v1 = t & 255, v2 = (t >> 8) & 255, l = t >> 16;
        const double* a1 = As + v1 * L2 + l * l;
        const double* a2 = As + v2 * L2 + l * l;
        double b = 0.0;
        for (int i = 0; i <= 2 * l; i++) b = fma(a1[i], a2[i], b);
        n2 = fma(b, b, n2);
    }
    n2 = warp_sum(n2);
    const double nrm = sqrt(n2);
    const double inv = (nrm > 0.0) ? 1.0 / nrm : 0.0;  // empty neighbourhood: B^ = 0 (R8)
    const int orow = out_map ? out_map[k] : local;
    double* brow = bh_out + (size_t)orow * ld;
    const int pend = min(gd.K, ld);
    for (int p = lane; p < pend; p += 32) {
        double b = 0.0;
        if (p < gd.P) {
            const int t = __ldg(gd.table + p);
            const int v1 = t & 255, v2 = (t >> 8) & 255, l = t >> 16;
            const double* a1 = As + v1 * L2 + l * l;
            const double* a2 = As + v2 * L2 + l * l;
            for (int i = 0; i <= 2 * l; i++) b = fma(a1[i], a2[i], b);
        }
        brow[p] = b * inv;
    }
    if (lane == 0) nrm_out[orow] = nrm;
}

template <int LMAX>
static void launch_descriptor(Launcher& L, const Grid& g, const Basis& bs, const YNorm& yn, const Workspace& ws,
                              int mmax, const GroupDev* groups, int row0, int nrows, double* bh_out, int ld,
                              double* nrm_out, const int* out_map, bool write_A) {
    constexpr int L2 = (LMAX + 1) * (LMAX + 1);
    const size_t smem = sizeof(double) * kDescWarps * (size_t)desc_warp_doubles(bs.n_max, L2, bs.NvL2);
    static size_t configured = 0;
    if (smem > 48 * 1024 && smem > configured) {
        cudaFuncSetAttribute(k_descriptor<LMAX>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        configured = smem;
    }
    L.launch(k_descriptor<LMAX>, dim3((nrows + kDescWarps - 1) / kDescWarps), dim3(kDescWarps * 32), smem, g, bs, yn,
             (const AtomS*)ws.atoms, (const int*)ws.nbr_cnt, (const int*)ws.nbr_idx, mmax, (const int*)ws.atom_of_row,
             (const unsigned char*)ws.gid, groups, row0, nrows, write_A ? ws.A : (double*)nullptr, bh_out, ld, nrm_out,
             out_map);
}

void run_descriptors(Launcher& L, const Grid& g, const Basis& bs, const YNorm& yn, const Workspace& ws, int mmax,
                     const GroupDev* groups, int row0, int nrows, double* bh_out, int ld, double* nrm_out,
                     const int* out_map, bool write_A) {
    if (nrows <= 0) return;
    switch (bs.l_max) {
#define FLARE_CASE(LM) \
    case LM: launch_descriptor<LM>(L, g, bs, yn, ws, mmax, groups, row0, nrows, bh_out, ld, nrm_out, out_map, write_A); break;
        FLARE_CASE(0) FLARE_CASE(1) FLARE_CASE(2) FLARE_CASE(3) FLARE_CASE(4) FLARE_CASE(5) FLARE_CASE(6)
#undef FLARE_CASE
        default: break;
    }
}

}  // namespace flare
