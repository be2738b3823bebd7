// descriptor.cu -- steps a2 + a3: per-pair basis, A accumulation, B2 contraction.
// One launch per (chunk, group); a group's atoms share the set of neighbour species, so the
// whole launch works on the group's Nc = nsp * n_max compact radial channels.
//
// A warp owns kDescTA consecutive rows (atoms) and walks over the concatenation of their
// neighbour lists in passes of 32 pairs, one pair per lane, so that the transcendental work
// (rsqrt, cospi, Chebyshev and Y_lm recurrences) runs with nearly full lanes although one atom
// has only 12-18 neighbours:
//   1. stage: lane p evaluates g~_n and Y_lm of its pair and writes them, pair-contiguous, into
//      shared memory ([n][pair] and [lm][pair], row stride 36: conflict-free fragment loads);
//   2. accumulate: for every atom with pairs in the pass, A[cnu,lm] += sum_j [s_j = s] g~_n(j) Y_lm(j)
//      as an [Nc x M].[M x L^2] product on the FP64 tensor pipe (mma.sync m8n8k4), the species
//      selection folded into the A-operand;
//   3. finalize (when the atom's last pair has been consumed): A -> global (for the back-propagation),
//      B[cnu1 <= cnu2, l] = sum_m A[cnu1,l,m] A[cnu2,l,m] as per-l [Nc x (2l+1)].[(2l+1) x Nc] products on
//      the tensor pipe, stored straight from the accumulator fragments (the L values of one (cnu1,cnu2)
//      pair are contiguous), and ||B||.  B is stored UNNORMALISED: d^ = B/||B|| is applied by the
//      consumers (E = B^T beta B / ||B||^2), which saves a second pass over the row.
#include <algorithm>

#include "kernels.cuh"

namespace flare {

constexpr int kDescWarps = 4;
constexpr int kDescTA = 8;  // atoms per warp (upper bound; small systems take fewer, see launch_descriptor)
constexpr int kPS = 36;     // pair stride of the staged rows (= 4 mod 16)

__host__ __device__ constexpr int pad4mod16(int n) {  // smallest m >= n with m % 16 == 4
    return ((n + 11) / 16) * 16 + 4;
}

template <int LMAX, int NMAXP>
struct DescSmem {
    static constexpr int L2 = (LMAX + 1) * (LMAX + 1);
    static constexpr int YR = ((L2 + 7) / 8) * 8;  // Y rows incl. zero padding up to a multiple of 8
    static constexpr int AS = pad4mod16(YR);       // row stride of A (conflict-free operand loads)
    __host__ __device__ static int warp_doubles(int Nc8) { return NMAXP * kPS + YR * kPS + Nc8 * AS + 16; }
};

__device__ __forceinline__ void dmma884_d(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}

template <int LMAX, int NMAXP>
__global__ void __launch_bounds__(kDescWarps * 32)
k_descriptor(Grid g, Basis bs, YNorm yn, GroupRun gr, int ta, const AtomS* __restrict__ atoms, const int* __restrict__ nbr_cnt,
             const int* __restrict__ nbr_idx, int mmax, const int* __restrict__ atom_of_row,
             const int* __restrict__ group_start, double* __restrict__ A_out, double* __restrict__ b_out, int ld,
             double* __restrict__ nrm_out) {
    using SM = DescSmem<LMAX, NMAXP>;
    constexpr int L = LMAX + 1;
    constexpr int L2 = L * L;
    constexpr int NBY = SM::YR / 8;
    constexpr int AS = SM::AS;
    extern __shared__ __align__(16) double smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    // rows of this group inside the chunk
    const int gs_ = max(group_start[gr.g], gr.row0);
    const int ge_ = min(group_start[gr.g + 1], gr.row0 + gr.nrows);
    const int g8 = lane >> 2, t4 = lane & 3;
    const int n_max = bs.n_max;
    const int Nc = gr.Nc, Nc8 = (Nc + 7) & ~7, nmb = Nc8 >> 3;
    double* gsm = smem + (size_t)warp * SM::warp_doubles(Nc8);  // [NMAXP][kPS]
    double* ysm = gsm + NMAXP * kPS;                             // [YR][kPS]
    double* As = ysm + SM::YR * kPS;                             // [Nc8][AS]
    int* sjs = reinterpret_cast<int*>(As + Nc8 * AS);            // [32] compact species of the staged pairs
    const bool one_species = gr.nsp == 1;
    // zeroed once per warp: the staged rows keep finite values from then on (idle lanes' columns are masked by a zero
    // operand, which needs a finite partner), the Y padding rows stay zero, and the first segment of an atom overwrites A
    if ((blockIdx.x * kDescWarps + warp) * ta < ge_ - gs_)
        for (int c = lane; c < (NMAXP + SM::YR) * kPS + Nc8 * AS; c += 32) gsm[c] = 0.0;
    // the grid is capped (a launch for a group with few or no rows costs next to nothing): a warp strides over its blocks
    for (int r0 = (blockIdx.x * kDescWarps + warp) * ta; r0 < ge_ - gs_; r0 += gridDim.x * kDescWarps * ta) {
    // warps are independent: only __syncwarp below
    const int na = min(ta, ge_ - gs_ - r0);
    const int lrow0 = gs_ - gr.row0 + r0;  // chunk-local row of the warp's first atom

    // per-lane atom bookkeeping (lanes 0..na-1), inclusive scan of the neighbour counts
    int my_k = 0, my_cnt = 0;
    if (lane < na) {
        my_k = atom_of_row[gs_ + r0 + lane];
        my_cnt = nbr_cnt[my_k];
    }
    int my_end = my_cnt;
#pragma unroll
    for (int o = 1; o < kDescTA; o <<= 1) {
        const int v = __shfl_up_sync(kFull, my_end, o);
        if (lane >= o) my_end += v;
    }
    const int my_start = my_end - my_cnt;
    const int T = __shfl_sync(kFull, my_end, kDescTA - 1);
    __syncwarp();

    // the loads of a pass are issued ahead of their use: the neighbour INDEX of pass q+2 and the two ATOMS of pass q+1
    // are requested during pass q (the kernel is otherwise stalled on these dependent, scattered 32-byte reads)
    auto locate = [&](int p, int& k, int& s) {
        int ai = 0;
#pragma unroll
        for (int i = 0; i < kDescTA - 1; i++) ai += (p >= __shfl_sync(kFull, my_end, i)) ? 1 : 0;
        k = __shfl_sync(kFull, my_k, ai);
        s = p - __shfl_sync(kFull, my_start, ai);
    };
    int k_n, s_n, j_n = 0, k_nn, s_nn, j_nn = 0;
    locate(lane, k_n, s_n);
    if (lane < T) j_n = nbr_idx[(size_t)k_n * mmax + s_n];
    locate(lane + 32, k_nn, s_nn);
    if (lane + 32 < T) j_nn = nbr_idx[(size_t)k_nn * mmax + s_nn];
    AtomS me_n = load_atom(atoms + k_n), o_n = load_atom(atoms + j_n);

    int a = 0;
    for (int p0 = 0;; p0 += 32) {
        // ---- 1. stage the basis of pairs [p0, p0+32)
        if (p0 < T) {
            const int p = p0 + lane;
            const AtomS me = me_n, o = o_n;
            if (p0 + 32 < T) {  // uniform
                k_n = k_nn; j_n = j_nn;
                me_n = load_atom(atoms + k_n);
                o_n = load_atom(atoms + j_n);
                if (p0 + 64 < T) {  // uniform
                    locate(p + 64, k_nn, s_nn);
                    j_nn = (p + 64 < T) ? nbr_idx[(size_t)k_nn * mmax + s_nn] : 0;
                }
            }
            int sj = -1;
            if (p < T) {
                double dx, dy, dz;
                displacement(g, me, o, dx, dy, dz);
                const double r2 = dx * dx + dy * dy + dz * dz;
                const double ir = rsqrt(r2);
                const double r = r2 * ir;
                sj = (int)((gr.sidx >> (4 * o.type)) & 15u);
                const double q = r * bs.irc[me.type * bs.S + o.type];
                const double x = 2.0 * q - 1.0;
                const double fc = 0.5 + 0.5 * cospi(q);
                double t0 = fc, t1 = x * fc;  // T_n(x) f_c
                const double x2 = 2.0 * x;
#pragma unroll
                for (int n = 0; n < NMAXP; n++) {
                    if (n < n_max) gsm[n * kPS + lane] = t0;
                    const double t2 = x2 * t1 - t0;
                    t0 = t1; t1 = t2;
                }
                real_ylm<LMAX, false>(yn, dx * ir, dy * ir, dz * ir,
                                      [&](int lm, double Y, double, double, double) { ysm[lm * kPS + lane] = Y; });
            }
            sjs[lane] = sj;
        }
        __syncwarp();
        // ---- 2./3. consume: every atom with pairs in this pass, in order
        while (a < na) {
            const int a_start = __shfl_sync(kFull, my_start, a);
            const int a_end = __shfl_sync(kFull, my_end, a);
            const int s0 = max(a_start, p0) - p0, s1 = min(a_end, p0 + 32) - p0;
            if (s1 > s0) {
                // A += G^T Y.  Fragment roles (m8n8k4): A-operand (row cnu = 8mb+g8, col j = k0+t4),
                // B-operand (row j = k0+t4, col lm = 8nb+g8), C (row cnu = 8mb+g8, cols lm = 8nb+2t4, +1).
                for (int mb = 0; mb < nmb; mb++) {
                    const int cnu = mb * 8 + g8;
                    int s_nu = -2, n_nu = 0;  // species block and radial index of the channel (no division)
                    if (cnu < Nc) {
                        s_nu = 0; n_nu = cnu;
                        while (n_nu >= n_max) { n_nu -= n_max; s_nu++; }
                    }
                    const double* grow = gsm + n_nu * kPS;
                    double acc[NBY][2];
#pragma unroll
                    for (int nb = 0; nb < NBY; nb++) { acc[nb][0] = 0.0; acc[nb][1] = 0.0; }
                    for (int k0 = s0 & ~3; k0 < s1; k0 += 4) {
                        const int j = k0 + t4;
                        // one neighbour species in the group: every pair feeds every channel (no species lookup)
                        const bool on = (j >= s0) && (j < s1) && (one_species ? s_nu == 0 : sjs[j] == s_nu);
                        const double av = on ? grow[j] : 0.0;
#pragma unroll
                        for (int nb = 0; nb < NBY; nb++)
                            dmma884_d(acc[nb][0], acc[nb][1], av, ysm[(nb * 8 + g8) * kPS + j]);
                    }
                    // the first segment of an atom overwrites A (nothing to re-zero between atoms); only an atom that
                    // continues from the previous pass accumulates
                    double* arow = As + cnu * AS + 2 * t4;
                    const bool first_seg = a_start >= p0;
#pragma unroll
                    for (int nb = 0; nb < NBY; nb++) {
                        double2* dst = reinterpret_cast<double2*>(arow + nb * 8);
                        double2 v = make_double2(acc[nb][0], acc[nb][1]);
                        if (!first_seg) { const double2 o = *dst; v.x += o.x; v.y += o.y; }
                        *dst = v;
                    }
                }
                __syncwarp();
            } else if (a_end == a_start) {  // an atom without neighbours (cannot be in a group with P > 0; kept for safety)
                for (int c = lane; c < Nc8 * AS; c += 32) As[c] = 0.0;
                __syncwarp();
            }
            if (a_end > p0 + 32) break;  // the atom continues in the next pass
            // ---- finalize atom a
            const int lrow = lrow0 + a;
            if (A_out) {
                double* arow = A_out + (size_t)lrow * bs.NvL2;
                if constexpr (L2 % 2 == 0) {
                    for (int c = 2 * lane; c < Nc * L2; c += 64) {
                        const int nu = c / L2;
                        *reinterpret_cast<double2*>(arow + c) = *reinterpret_cast<const double2*>(As + nu * AS + (c - nu * L2));
                    }
                } else {
                    for (int c = lane; c < Nc * L2; c += 32) {
                        const int nu = c / L2;
                        arow[c] = As[nu * AS + (c - nu * L2)];
                    }
                }
            }
            double* brow = b_out + (size_t)lrow * ld;
            double n2 = 0.0;
            for (int mb = 0; mb < nmb; mb++) {
                const int nu1 = mb * 8 + g8;
                const double* a1 = As + nu1 * AS + t4;
                for (int nb = mb; nb < nmb; nb++) {
                    const double* a2 = As + (nb * 8 + g8) * AS + t4;
                    double acc[L][2];
#pragma unroll
                    for (int l = 0; l < L; l++) {
                        acc[l][0] = 0.0; acc[l][1] = 0.0;
#pragma unroll
                        for (int ks = 0; ks < (2 * l + 1 + 3) / 4; ks++) {
                            const bool ok = 4 * ks + t4 < 2 * l + 1;
                            const double av = ok ? a1[l * l + 4 * ks] : 0.0;
                            const double bv = ok ? a2[l * l + 4 * ks] : 0.0;
                            dmma884_d(acc[l][0], acc[l][1], av, bv);
                        }
                    }
#pragma unroll
                    for (int e = 0; e < 2; e++) {
                        const int nu2 = nb * 8 + 2 * t4 + e;
                        if (nu1 <= nu2 && nu2 < Nc) {
                            // triangular enumeration over the compact channels (R4 order restricted to the group)
                            const int q = nu1 * Nc - (nu1 * (nu1 - 1)) / 2 + (nu2 - nu1);
                            double* dst = brow + (size_t)q * L;
#pragma unroll
                            for (int l = 0; l < L; l++) n2 = fma(acc[l][e], acc[l][e], n2);
                            if constexpr (L % 2 == 0) {
#pragma unroll
                                for (int l = 0; l < L; l += 2)
                                    *reinterpret_cast<double2*>(dst + l) = make_double2(acc[l][e], acc[l + 1][e]);
                            } else {
#pragma unroll
                                for (int l = 0; l < L; l++) dst[l] = acc[l][e];
                            }
                        }
                    }
                }
            }
            n2 = warp_sum(n2);
            for (int p = gr.P + lane; p < gr.K; p += 32) brow[p] = 0.0;  // zero padding up to K
            if (lane == 0) nrm_out[lrow] = n2;  // ||B||^2 (the consumers need 1/||B||^2); no neighbours: 0 (R8)
            __syncwarp();
            a++;
        }
        __syncwarp();
        if (a >= na) break;
    }
    __syncwarp();
    }  // blocks of this warp
}

template <int LMAX, int NMAXP>
static void launch_descriptor(Launcher& L, const Grid& g, const Basis& bs, const YNorm& yn, const Workspace& ws,
                              int mmax, const GroupRun& gr, double* bh_out, int ld, double* nrm_out, bool write_A) {
    using SM = DescSmem<LMAX, NMAXP>;
    const int Nc8 = (gr.Nc + 7) & ~7;
    const size_t smem = sizeof(double) * kDescWarps * (size_t)SM::warp_doubles(Nc8);
    L.ensure_smem(k_descriptor<LMAX, NMAXP>, smem);
    const int ta = small_system_ta(gr.nrows, kDescWarps, kDescTA);
    const int per_cta = kDescWarps * ta;
    const int grid = std::min((gr.nrows + per_cta - 1) / per_cta, 148 * 32);
    L.launch(k_descriptor<LMAX, NMAXP>, dim3(grid), dim3(kDescWarps * 32), smem, g, bs, yn,
             gr, ta, (const AtomS*)ws.atoms, (const int*)ws.nbr_cnt, (const int*)ws.nbr_idx, mmax,
             (const int*)ws.atom_of_row, (const int*)ws.group_start, write_A ? ws.A : (double*)nullptr, bh_out, ld,
             nrm_out);
}

void run_descriptors(Launcher& L, const Grid& g, const Basis& bs, const YNorm& yn, const Workspace& ws, int mmax,
                     const GroupDesc* groups, int n_groups, int row0, int nrows, double* bh_out, int ld,
                     double* nrm_out, bool write_A) {
    if (nrows <= 0) return;
    L.fork();
    for (int gi = 0; gi < n_groups; gi++) {
        if (groups[gi].P == 0) continue;  // no neighbours: no descriptor (R8); nothing downstream reads these rows
        const GroupRun gr = make_group_run(groups[gi], gi, row0, nrows);
        L.select(gi);
#define FLARE_CASE(LM)                                                                                   \
    case LM:                                                                                             \
        if (bs.n_max <= 8) launch_descriptor<LM, 8>(L, g, bs, yn, ws, mmax, gr, bh_out, ld, nrm_out, write_A);       \
        else if (bs.n_max <= 10) launch_descriptor<LM, 10>(L, g, bs, yn, ws, mmax, gr, bh_out, ld, nrm_out, write_A); \
        else if (bs.n_max <= 12) launch_descriptor<LM, 12>(L, g, bs, yn, ws, mmax, gr, bh_out, ld, nrm_out, write_A); \
        else launch_descriptor<LM, 16>(L, g, bs, yn, ws, mmax, gr, bh_out, ld, nrm_out, write_A);                    \
        break;
        switch (bs.l_max) {
            FLARE_CASE(0) FLARE_CASE(1) FLARE_CASE(2) FLARE_CASE(3) FLARE_CASE(4) FLARE_CASE(5) FLARE_CASE(6)
            default: break;
        }
#undef FLARE_CASE
    }
    L.join();
}

}  // namespace flare
