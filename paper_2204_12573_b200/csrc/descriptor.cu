// descriptor.cu -- steps a2 + a3: per-pair basis, A accumulation, B2 contraction, normalisation
// (P:L123-129).  One warp per atom:
//   1. neighbours are spread across lanes for the basis evaluation (sqrt, sincospi, Chebyshev and
//      Y_lm recurrences); g~_n and Y_lm of up to 32 neighbours are staged in shared memory;
//   2. A[nu,lm] = sum_j [s_j = s] g~_n(j) Y_lm(j) is a small dense contraction over the neighbours
//      (an [N_nu x M] . [M x L^2] product); it runs on the FP64 tensor pipe (mma.sync m8n8k4) with
//      the species selection folded into the A-operand, so no shuffle reduction over the 256+
//      components and no per-component shared-memory loop is needed;
//   3. B[nu1<=nu2, l] = sum_m A[nu1,l,m] A[nu2,l,m]: one (nu1,nu2) pair per lane, all l at once, so a
//      warp writes 32 x (l_max+1) consecutive doubles of the B^ row (fully coalesced); two passes
//      (norm, then scaled store) recompute the cheap contraction instead of holding B in registers.
#include "kernels.cuh"

namespace flare {

constexpr int kDescWarps = 4;

__host__ __device__ inline int desc_warp_doubles(int n_max, int L2, int Nv) {
    // g[32][n_max|1], Y[32][L2|1], A[Nv][L2|1], species[32] (ints, 16 doubles)
    return 32 * (n_max | 1) + 32 * (L2 | 1) + Nv * (L2 | 1) + 16;
}

__device__ __forceinline__ void dmma884_d(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}

template <int LMAX>
__global__ void __launch_bounds__(kDescWarps * 32)
k_descriptor(Grid g, Basis bs, YNorm yn, const AtomS* __restrict__ atoms, const int* __restrict__ nbr_cnt,
             const int* __restrict__ nbr_idx, int mmax, const int* __restrict__ atom_of_row,
             const unsigned char* __restrict__ gid, const GroupDev* __restrict__ groups, int row0, int nrows,
             double* __restrict__ A_out, double* __restrict__ bh_out, int ld, double* __restrict__ nrm_out,
             const int* __restrict__ out_map) {
    constexpr int L = LMAX + 1;
    constexpr int L2 = L * L;
    constexpr int YS = L2 | 1;  // odd row strides: conflict-free column access across rows
    constexpr int AS = L2 | 1;
    extern __shared__ double smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int local = blockIdx.x * kDescWarps + warp;
    if (local >= nrows) return;  // warps are independent: only __syncwarp below
    const int g8 = lane >> 2, t4 = lane & 3;
    const int GS = bs.n_max | 1;
    const int Nv = bs.Nv;
    double* gs = smem + (size_t)warp * desc_warp_doubles(bs.n_max, L2, Nv);
    double* ys = gs + 32 * GS;
    double* As = ys + 32 * YS;
    int* sjs = reinterpret_cast<int*>(As + Nv * AS);

    const int k = atom_of_row[row0 + local];
    const AtomS me = load_atom(atoms + k);
    const int cnt = nbr_cnt[k];
    for (int c = lane; c < Nv * AS; c += 32) As[c] = 0.0;

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
        // A += G^T Y on the tensor pipe.  Fragment roles (m8n8k4): A-operand (row nu = 8mb+g8, col j = k0+t4),
        // B-operand (row j = k0+t4, col lm = 8nb+g8), C (row nu = 8mb+g8, cols lm = 8nb+2t4, +1).
        for (int mb = 0; mb * 8 < Nv; mb++) {
            const int nu = mb * 8 + g8;
            const int s_nu = (nu < Nv) ? nu / bs.n_max : -2;
            const int n_nu = nu - s_nu * bs.n_max;
#pragma unroll 1
            for (int nb = 0; nb * 8 < L2; nb++) {
                const int lmb = nb * 8 + g8;
                double c0 = 0.0, c1 = 0.0;
                for (int k0 = 0; k0 < nact; k0 += 4) {
                    const int j = k0 + t4;  // < 32 always; lanes >= nact carry sjs = -1
                    const double a = (sjs[j] == s_nu) ? gs[j * GS + n_nu] : 0.0;
                    const double b = (j < nact && lmb < L2) ? ys[j * YS + lmb] : 0.0;
                    dmma884_d(c0, c1, a, b);
                }
                const int lm0 = nb * 8 + 2 * t4;
                if (nu < Nv) {
                    if (lm0 < L2) As[nu * AS + lm0] += c0;
                    if (lm0 + 1 < L2) As[nu * AS + lm0 + 1] += c1;
                }
            }
        }
        __syncwarp();
    }

    if (A_out) {
        double* arow = A_out + (size_t)local * bs.NvL2;
        for (int c = lane; c < bs.NvL2; c += 32) {
            const int nu = c / L2;
            arow[c] = As[nu * AS + (c - nu * L2)];
        }
    }

    // B2 contraction, one (nu1,nu2) pair per lane, all l at once.
    const GroupDev gd = groups[gid[k]];
    const int npairs = gd.P / L;
    double n2 = 0.0;
    for (int q = lane; q < npairs; q += 32) {
        const int t = __ldg(gd.table + q);
        const double* a1 = As + (t & 255) * AS;
        const double* a2 = As + (t >> 8) * AS;
#pragma unroll
        for (int l = 0; l < L; l++) {
            double b = 0.0;
#pragma unroll
            for (int i = l * l; i < (l + 1) * (l + 1); i++) b = fma(a1[i], a2[i], b);
            n2 = fma(b, b, n2);
        }
    }
    n2 = warp_sum(n2);
    const double nrm = sqrt(n2);
    const double inv = (nrm > 0.0) ? 1.0 / nrm : 0.0;  // empty neighbourhood: B^ = 0 (R8)
    const int orow = out_map ? out_map[k] : local;
    double* brow = bh_out + (size_t)orow * ld;
    for (int q = lane; q < npairs; q += 32) {
        const int t = __ldg(gd.table + q);
        const double* a1 = As + (t & 255) * AS;
        const double* a2 = As + (t >> 8) * AS;
#pragma unroll
        for (int l = 0; l < L; l++) {
            double b = 0.0;
#pragma unroll
            for (int i = l * l; i < (l + 1) * (l + 1); i++) b = fma(a1[i], a2[i], b);
            brow[q * L + l] = b * inv;
        }
    }
    for (int p = gd.P + lane; p < min(gd.K, ld); p += 32) brow[p] = 0.0;  // zero padding up to K
    if (lane == 0) nrm_out[orow] = nrm;
}

template <int LMAX>
static void launch_descriptor(Launcher& L, const Grid& g, const Basis& bs, const YNorm& yn, const Workspace& ws,
                              int mmax, const GroupDev* groups, int row0, int nrows, double* bh_out, int ld,
                              double* nrm_out, const int* out_map, bool write_A) {
    constexpr int L2 = (LMAX + 1) * (LMAX + 1);
    const size_t smem = sizeof(double) * kDescWarps * (size_t)desc_warp_doubles(bs.n_max, L2, bs.Nv);
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
