// force.cu -- steps a6 + a7: back-propagation of dE/dB through A to per-pair forces, and the
// atomics-free force gather ("reordering the summation" so that grad d_i is never formed).
//
// k_backprop, one launch per (chunk, group), a warp per block of up to 8 rows (atoms) k:
//   E_k   = sum of the energy tiles' partial row-dots (fixed order) / ||B||^2     (Eq. 1; rows hold unnormalised B)
//   V_k   = same for the variance tiles                                            (Eq. 2)
//   c_p   = dE_k/dB_p = (2/||B||^2)(W_p - E_k B_p),  W = beta B                   (R10, R11)
//   G[nu1,lm] = dE_k/dA[nu1,lm] = sum_{nu2} c_{p(nu1,nu2,l)} (1+delta) A[nu2,lm]   (FP64 tensor pipe)
//   f_kj  = dE_k/dr_kj = sum_{n,lm} G[s_j n, lm] grad(g~_n Y_lm)(r_kj)   for every neighbour j, one pair per lane over
//           the concatenated neighbour lists of the warp's atoms
// f_kj is stored once per ordered pair.  k_gather then forms, with the reverse-pair index,
//   F_k = sum_j ( f_kj - f_jk )
// reading each pair force exactly twice and writing each atom's force exactly once.
#include <algorithm>

#include "kernels.cuh"

namespace flare {

constexpr int kBpWarps = 4;
constexpr int kBpMaxTA = 8;  // atoms per warp (upper bound; the launch picks ta <= 8 from the shared-memory budget)

__host__ __device__ constexpr int bp_pad4mod16(int n) { return ((n + 11) / 16) * 16 + 4; }

template <int LMAX, int NMAXP>
struct BpSmem {
    static constexpr int L2 = (LMAX + 1) * (LMAX + 1);
    static constexpr int AS = bp_pad4mod16(L2);    // row stride of the staged A (conflict-free operand loads)
    static constexpr int GB = L2 * NMAXP + 2;      // G^T block of one (atom, species): [L2][NMAXP] + bank shift
    // G^T of ta atoms + double-buffered [A | W | B] rows of one atom (filled by cp.async one atom ahead)
    // staged: W and B rows go through shared memory too (small K); otherwise only A does and dE/dB is formed from global
    // memory (large K: the rows would cost resident warps)
    __host__ __device__ static int warp_doubles(int ta, int nsp, int Nc8, int K, bool staged) {
        return (ta * nsp * GB + 2 * (Nc8 * AS + (staged ? 2 * K : 0)) + 1) & ~1;  // even: 16-byte aligned regions
    }
};

__device__ __forceinline__ void bp_cp_async16(void* smem_dst, const void* gmem_src) {
    unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(d), "l"(gmem_src));
}
__device__ __forceinline__ void bp_cp_async8(void* smem_dst, const void* gmem_src) {
    unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"(d), "l"(gmem_src));
}

__device__ __forceinline__ void dmma884_f(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}

// g[n] = T_n(x) f_c(r), dg[n] = d g[n]/dr for n < n_max, zero above; fully unrolled so that g/dg stay in registers
template <int NMAXP>
__device__ __forceinline__ void radial_fixed(int n_max, double r, double inv_rc, double (&gv)[NMAXP],
                                             double (&dgv)[NMAXP]) {
    const double q = r * inv_rc;
    const double x = 2.0 * q - 1.0;
    double sn, cs;
    sincospi(q, &sn, &cs);
    const double fc = 0.5 + 0.5 * cs;
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

// One launch per (chunk, group).  A warp owns `ta` consecutive rows: phase 1 forms E, V, c = dE/dB and
// G = dE/dA of each of its atoms (G on the tensor pipe), phase 2 walks over the concatenated neighbour
// lists of those atoms, one pair per lane, so that the basis gradients run with nearly full lanes.
template <int LMAX, int NMAXP, bool STAGED>
__global__ void __launch_bounds__(kBpWarps * 32, 4)
k_backprop(Grid g, Basis bs, YNorm yn, GroupRun gr, int ta, const AtomS* __restrict__ atoms,
           const int* __restrict__ nbr_cnt, const int* __restrict__ nbr_idx, int mmax,
           const int* __restrict__ atom_of_row, const int* __restrict__ group_start, const double* __restrict__ A_in,
           const double* __restrict__ Braw, const double* __restrict__ W, const double* __restrict__ nrm_in,
           const double* __restrict__ part, int ld, int chunk_cap, int max_ntn, int want_variance,
           double* __restrict__ pairf, double* __restrict__ e_s, double* __restrict__ v_s) {
    using SM = BpSmem<LMAX, NMAXP>;
    constexpr int L = LMAX + 1;
    constexpr int L2 = L * L;
    constexpr int AS = SM::AS;
    constexpr int GB = SM::GB;
    constexpr int NBL = (2 * LMAX + 1 + 7) / 8;  // n8 blocks needed for the widest m range
    extern __shared__ __align__(16) double smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int gs_ = max(group_start[gr.g], gr.row0);
    const int ge_ = min(group_start[gr.g + 1], gr.row0 + gr.nrows);
    // 1..kBpWarps warps per CTA (shared-memory budget); the grid is capped (a launch for a group with few or no rows
    // costs next to nothing): a warp strides over its blocks.  Warps are independent: only __syncwarp below.
    const int wpc = blockDim.x >> 5;
    for (int r0 = (blockIdx.x * wpc + warp) * ta; r0 < ge_ - gs_; r0 += gridDim.x * wpc * ta) {
    const int na = min(ta, ge_ - gs_ - r0);
    const int lrow0 = gs_ - gr.row0 + r0;
    const int g8 = lane >> 2, t4 = lane & 3;
    const int n_max = bs.n_max;
    const int Nc = gr.Nc, Nc8 = (Nc + 7) & ~7, nmb = Nc8 >> 3;
    double* Gt = smem + (size_t)warp * SM::warp_doubles(ta, gr.nsp, Nc8, gr.K, STAGED);  // [ta][nsp][GB]
    double* rows = Gt + ta * gr.nsp * GB;  // [2][ A [Nc8][AS] | W [K] | B [K] ]
    const int row_doubles = Nc8 * AS + (STAGED ? 2 * gr.K : 0);
    // the first loads of the block are issued before anything else: the atom of each row, and (lane a for atom a) the
    // first tile partials and ||B|| that phase 1 starts from
    int my_k = 0, my_cnt = 0;
    double pE0 = 0.0, pV0 = 0.0, pnrm = 0.0;
    if (lane < na) {
        my_k = atom_of_row[gs_ + r0 + lane];
        if (gr.ntn > 0) {
            pE0 = part[lrow0 + lane];
            if (want_variance) pV0 = part[(size_t)max_ntn * chunk_cap + lrow0 + lane];
        }
        if (gr.P > 0) pnrm = nrm_in[lrow0 + lane];
    }
    // what is read without having been written: G^T rows n >= n_max (B operand of the pair phase) and the A rows of the
    // padding channels Nc .. Nc8 (multiplied by a zero dE/dB, but 0 x NaN would poison the accumulator)
    if (n_max < NMAXP)
        for (int c = lane; c < ta * gr.nsp * GB; c += 32) Gt[c] = 0.0;
    if (Nc < Nc8)
        for (int c = lane; c < 2 * (Nc8 - Nc) * AS; c += 32) {
            const int buf = c / ((Nc8 - Nc) * AS);
            rows[buf * row_doubles + Nc * AS + (c - buf * (Nc8 - Nc) * AS)] = 0.0;
        }
    if (lane < na) my_cnt = nbr_cnt[my_k];
    int my_end = my_cnt;
#pragma unroll
    for (int o = 1; o < kBpMaxTA; o <<= 1) {
        const int v = __shfl_up_sync(kFull, my_end, o);
        if (lane >= o) my_end += v;
    }
    const int my_start = my_end - my_cnt;
    const int T = __shfl_sync(kFull, my_end, kBpMaxTA - 1);
    __syncwarp();

    // Phase-2 loads (neighbour index, then the two atoms) are issued one pass ahead of their use; the first
    // pass's already here, so that they fly during phase 1.
    auto locate = [&](int p, int& ai, int& k, int& s) {
        ai = 0;
#pragma unroll
        for (int i = 0; i < kBpMaxTA - 1; i++) ai += (p >= __shfl_sync(kFull, my_end, i)) ? 1 : 0;
        k = __shfl_sync(kFull, my_k, ai);
        s = p - __shfl_sync(kFull, my_start, ai);
    };
    // pipeline depth 2: the neighbour INDEX of pass q+2 and the two ATOMS of pass q+1 are requested during pass q,
    // so that neither the index -> atom dependency nor the atom loads themselves stall a pass
    int ai_n, k_n, s_n, j_n = 0;
    locate(lane, ai_n, k_n, s_n);
    if (lane < T) j_n = nbr_idx[(size_t)k_n * mmax + s_n];
    int ai_nn, k_nn, s_nn, j_nn = 0;
    locate(lane + 32, ai_nn, k_nn, s_nn);
    if (lane + 32 < T) j_nn = nbr_idx[(size_t)k_nn * mmax + s_nn];
    AtomS me_n = load_atom(atoms + k_n), o_n = load_atom(atoms + j_n);

    // ---------------- phase 1: per atom E, V, c, G
    // E, V from the tile partials (fixed order => deterministic), lane a for atom a so that the loads of all
    // atoms are in flight together; the rows hold the unnormalised B, so E = B^T beta B / ||B||^2 and
    // c = dE/dB = (2/||B||^2)(W - E B) with W = beta B   (R10, R11)
    double my_E = 0.0, my_inv2 = 0.0;
    if (lane < na) {
        const int lrow = lrow0 + lane;
        double E = pE0, V = pV0;
        for (int t = 1; t < gr.ntn; t++) E += part[(size_t)t * chunk_cap + lrow];
        if (want_variance)
            for (int t = 1; t < gr.ntn; t++) V += part[((size_t)max_ntn + t) * chunk_cap + lrow];
        my_inv2 = (pnrm > 0.0) ? 1.0 / pnrm : 0.0;  // pnrm = ||B||^2; no neighbours: E = V = 0 (R8)
        my_E = E * my_inv2;
        e_s[my_k] = my_E;
        v_s[my_k] = V * my_inv2;
    }
    // A (compact, into its padded layout), W = beta B and B of one atom -> shared memory, asynchronously
    auto issue_rows = [&](int a, int buf) {
        const int lrow = lrow0 + a;
        double* As = rows + buf * row_doubles;
        const double* arow = A_in + (size_t)lrow * bs.NvL2;
        if constexpr (L2 % 2 == 0) {
            for (int c = 2 * lane; c < Nc * L2; c += 64) {
                const int nu = c / L2;
                bp_cp_async16(As + nu * AS + (c - nu * L2), arow + c);
            }
        } else {
            for (int c = lane; c < Nc * L2; c += 32) {
                const int nu = c / L2;
                bp_cp_async8(As + nu * AS + (c - nu * L2), arow + c);
            }
        }
        if constexpr (STAGED) {
            double* Ws = As + Nc8 * AS;
            const double* wrow = W + (size_t)lrow * ld;
            const double* brow = Braw + (size_t)lrow * ld;
            for (int c = 2 * lane; c < gr.K; c += 64) {
                bp_cp_async16(Ws + c, wrow + c);
                bp_cp_async16(Ws + gr.K + c, brow + c);
            }
        }
    };
    if (gr.P > 0) issue_rows(0, 0);
    asm volatile("cp.async.commit_group;\n" ::);
    for (int a = 0; a < na && gr.P > 0; a++) {
        if (a + 1 < na) issue_rows(a + 1, (a + 1) & 1);
        asm volatile("cp.async.commit_group;\n" ::);
        asm volatile("cp.async.wait_group 1;\n" ::);
        __syncwarp();
        const double E = __shfl_sync(kFull, my_E, a);
        const double two_inv2 = 2.0 * __shfl_sync(kFull, my_inv2, a);
        const double* As = rows + (a & 1) * row_doubles;
        // W and B of this atom: staged in shared memory, or (large K) read where they are, in global memory
        const double* Ws = STAGED ? As + Nc8 * AS : W + (size_t)(lrow0 + a) * ld;
        const double* Bs = STAGED ? Ws + gr.K : Braw + (size_t)(lrow0 + a) * ld;

        // G[cnu1, (l,m)] = sum_cnu2 C_l[cnu1,cnu2] A[cnu2,(l,m)], C_l[cnu1,cnu2] = c[q(cnu1,cnu2) L + l]: per l a small
        // symmetric-matrix product on the tensor pipe.  A-operand (row cnu1 = 8mb+g8, col cnu2 = k0+t4),
        // B-operand (row cnu2 = k0+t4, col m = 8nb+g8), C (row cnu1, cols m = 8nb+2t4, +1).
        double* Gta = Gt + (size_t)a * gr.nsp * GB;
        for (int mb = 0; mb < nmb; mb++) {
            const int nu1 = mb * 8 + g8;
            double acc[L][NBL][2];
#pragma unroll
            for (int l = 0; l < L; l++)
#pragma unroll
                for (int nb = 0; nb < NBL; nb++) { acc[l][nb][0] = 0.0; acc[l][nb][1] = 0.0; }
            for (int k0 = 0; k0 < Nc8; k0 += 4) {
                const int nu2 = k0 + t4;
                const bool in = nu1 < Nc && nu2 < Nc;
                const int lo = min(nu1, nu2), hi = max(nu1, nu2);
                const int cq = in ? (lo * Nc - (lo * (lo - 1)) / 2 + (hi - lo)) * L : 0;
                const double fac = (nu1 == nu2) ? 2.0 * two_inv2 : two_inv2;  // (1 + delta) of the diagonal pairs
                const double* a2 = As + nu2 * AS + g8;
                // the L values of W and B of this channel pair are contiguous: fetched with 16-byte loads (half the
                // shared-memory instructions, and the 8-byte loads at stride L were 4-way bank conflicts)
                double wv[L], bvv[L];
                if constexpr (L % 2 == 0) {
#pragma unroll
                    for (int l = 0; l < L; l += 2) {
                        const double2 w2 = *reinterpret_cast<const double2*>(Ws + cq + l);
                        const double2 b2 = *reinterpret_cast<const double2*>(Bs + cq + l);
                        wv[l] = w2.x; wv[l + 1] = w2.y; bvv[l] = b2.x; bvv[l + 1] = b2.y;
                    }
                } else {
#pragma unroll
                    for (int l = 0; l < L; l++) { wv[l] = Ws[cq + l]; bvv[l] = Bs[cq + l]; }
                }
#pragma unroll
                for (int l = 0; l < L; l++) {
                    const double av = in ? fac * (wv[l] - E * bvv[l]) : 0.0;  // c = dE/dB
#pragma unroll
                    for (int nb = 0; nb < NBL; nb++) {
                        if (nb * 8 < 2 * l + 1) {
                            const double bv = (nb * 8 + g8 < 2 * l + 1) ? a2[l * l + nb * 8] : 0.0;
                            dmma884_f(acc[l][nb][0], acc[l][nb][1], av, bv);
                        }
                    }
                }
            }
            if (nu1 < Nc) {
                int s1 = 0, n1 = nu1;  // species block of the channel (no division: at most nsp - 1 subtractions)
                while (n1 >= n_max) { n1 -= n_max; s1++; }
                double* gt = Gta + (size_t)s1 * GB + n1;
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
    }

    // ---------------- phase 2: per-pair forces f_kj = sum_{n,lm} G[s_j n, lm] grad(g~_n Y_lm)(r_kj), one pair per lane
    for (int p0 = 0; p0 < T; p0 += 32) {
        const int p = p0 + lane;
        const int ai = ai_n, k = k_n, s = s_n;
        const AtomS me = me_n, o = o_n;
        if (p0 + 32 < T) {  // uniform
            ai_n = ai_nn; k_n = k_nn; s_n = s_nn; j_n = j_nn;
            me_n = load_atom(atoms + k_n);
            o_n = load_atom(atoms + j_n);
            if (p0 + 64 < T) {  // uniform
                locate(p + 64, ai_nn, k_nn, s_nn);
                j_nn = (p + 64 < T) ? nbr_idx[(size_t)k_nn * mmax + s_nn] : 0;
            }
        }
        if (p < T) {
            double dx, dy, dz;
            displacement(g, me, o, dx, dy, dz);
            const double r2 = dx * dx + dy * dy + dz * dz;
            const double ir = rsqrt(r2);
            const double r = r2 * ir;
            const double ux = dx * ir, uy = dy * ir, uz = dz * ir;
            double gr_[NMAXP], dgr[NMAXP];
            radial_fixed<NMAXP>(n_max, r, bs.irc[me.type * bs.S + o.type], gr_, dgr);
            const int sj = (int)((gr.sidx >> (4 * o.type)) & 15u);
            const double* Gj = Gt + (size_t)(ai * gr.nsp + sj) * GB;
            double srad = 0.0, vx = 0.0, vy = 0.0, vz = 0.0;
            real_ylm<LMAX, true>(yn, ux, uy, uz, [&](int lm, double Y, double gx, double gy, double gz) {
                const double2* gp = reinterpret_cast<const double2*>(Gj + lm * NMAXP);
                // sum_n G[n,lm] dg_n  and  sum_n G[n,lm] g_n, as four independent chains
                double hr = 0.0, hg = 0.0, hr1 = 0.0, hg1 = 0.0;
#pragma unroll
                for (int n2 = 0; n2 < NMAXP / 2; n2++) {
                    const double2 Gv = gp[n2];
                    hr = fma(Gv.x, dgr[2 * n2], hr);
                    hr1 = fma(Gv.y, dgr[2 * n2 + 1], hr1);
                    hg = fma(Gv.x, gr_[2 * n2], hg);
                    hg1 = fma(Gv.y, gr_[2 * n2 + 1], hg1);
                }
                hr += hr1;
                hg += hg1;
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
    __syncwarp();
    }  // blocks of this warp
}

template <int LMAX, int NMAXP, bool STAGED>
static void launch_backprop_(Launcher& L, const Grid& g, const Basis& bs, const YNorm& yn, const Workspace& ws,
                            int mmax, const GroupRun& gr, int ld, int chunk_cap, int max_ntn, bool want_variance) {
    using SM = BpSmem<LMAX, NMAXP>;
    const int Nc8 = (gr.Nc + 7) & ~7;
    // atoms per warp (1..8) against resident CTAs per SM (1..4: 128 registers per thread): more atoms per warp pack more
    // pairs into each 32-lane pass, but their G^T blocks cost shared memory.  Take the most CTAs that still leave at
    // least two atoms per warp, and then as many atoms as fit (measured: (8,3) 4 CTAs x 6 atoms, (10,4) 4 x 2 beats
    // 2 x 7, (12,6) 2 x 3 beats 3 x 1).
    int ta = kBpMaxTA;
    if (gr.nsp > 0) {
        const size_t sm_bytes = 228 * 1024;  // per SM
        // + 1 KB: the shared memory the system reserves per resident CTA
        auto cta_bytes = [&](int t) { return sizeof(double) * kBpWarps * (size_t)SM::warp_doubles(t, gr.nsp, Nc8, gr.K, STAGED) + 1024; };
        auto fit = [&](int target) {
            int t = kBpMaxTA;
            while (t > 1 && cta_bytes(t) * target > sm_bytes) t--;
            return t;
        };
        int target = 4;
        while (target > 1 && (cta_bytes(1) * target > sm_bytes || fit(target) < 2)) target--;
        ta = fit(target);
    }
    ta = std::min(ta, small_system_ta(gr.nrows, kBpWarps, kBpMaxTA));
    // warps per CTA: as many of kBpWarps as fit the 227 KB of shared memory a CTA can have (large (n_max, l_max))
    const size_t per_warp = sizeof(double) * (size_t)SM::warp_doubles(ta, gr.nsp, Nc8, gr.K, STAGED);
    int warps = kBpWarps;
    while (warps > 1 && per_warp * warps > 220 * 1024) warps--;
    const size_t smem = per_warp * warps;
    if (smem > 227 * 1024) {
        if (L.err == cudaSuccess) { L.err = cudaErrorInvalidValue; L.err_where = "back-propagation: descriptor too large for shared memory"; }
        return;
    }
    L.ensure_smem(k_backprop<LMAX, NMAXP, STAGED>, smem);
    const int per_cta = warps * ta;
    const int grid = std::min((gr.nrows + per_cta - 1) / per_cta, 148 * 32);
    L.launch(k_backprop<LMAX, NMAXP, STAGED>, dim3(grid), dim3(warps * 32), smem, g, bs, yn, gr,
             ta, (const AtomS*)ws.atoms, (const int*)ws.nbr_cnt, (const int*)ws.nbr_idx, mmax,
             (const int*)ws.atom_of_row, (const int*)ws.group_start, (const double*)ws.A, (const double*)ws.Bh,
             (const double*)ws.W, (const double*)ws.nrm, (const double*)ws.part, ld, chunk_cap, max_ntn,
             want_variance ? 1 : 0, ws.pairf, ws.e_s, ws.v_s);
}

// W and B rows staged through shared memory only while they are small (K <= 160: the single-species groups of (8,3));
// for larger K the 2 x 2K doubles per warp would cost resident warps (one CTA of 4 warps per SM at (12,6))
template <int LMAX, int NMAXP>
static void launch_backprop(Launcher& L, const Grid& g, const Basis& bs, const YNorm& yn, const Workspace& ws,
                            int mmax, const GroupRun& gr, int ld, int chunk_cap, int max_ntn, bool want_variance) {
    if (gr.K <= 160) launch_backprop_<LMAX, NMAXP, true>(L, g, bs, yn, ws, mmax, gr, ld, chunk_cap, max_ntn, want_variance);
    else launch_backprop_<LMAX, NMAXP, false>(L, g, bs, yn, ws, mmax, gr, ld, chunk_cap, max_ntn, want_variance);
}

void run_backprop(Launcher& L, const Grid& g, const Basis& bs, const YNorm& yn, const Workspace& ws, int mmax,
                  const GroupDesc* groups, int n_groups, int row0, int nrows, int ld, int chunk_cap, int max_ntn,
                  bool want_variance) {
    if (nrows <= 0) return;
    L.fork();
    for (int gi = 0; gi < n_groups; gi++) {
        const GroupRun gr = make_group_run(groups[gi], gi, row0, nrows);
        L.select(gi);
#define FLARE_CASE(LM)                                                                                        \
    case LM:                                                                                                  \
        if (bs.n_max <= 8) launch_backprop<LM, 8>(L, g, bs, yn, ws, mmax, gr, ld, chunk_cap, max_ntn, want_variance);       \
        else if (bs.n_max <= 10) launch_backprop<LM, 10>(L, g, bs, yn, ws, mmax, gr, ld, chunk_cap, max_ntn, want_variance); \
        else if (bs.n_max <= 12) launch_backprop<LM, 12>(L, g, bs, yn, ws, mmax, gr, ld, chunk_cap, max_ntn, want_variance); \
        else launch_backprop<LM, 16>(L, g, bs, yn, ws, mmax, gr, ld, chunk_cap, max_ntn, want_variance);                    \
        break;
        switch (bs.l_max) {
            FLARE_CASE(0) FLARE_CASE(1) FLARE_CASE(2) FLARE_CASE(3) FLARE_CASE(4) FLARE_CASE(5) FLARE_CASE(6)
            default: break;
        }
#undef FLARE_CASE
    }
    L.join();
}

// ------------------------------------------------------------------ a7: atomics-free gather
constexpr int kGatherWarps = 8;
constexpr int kGatherAPW = 4;  // atoms per warp: 8 lanes each, so that a warp keeps ~3x more scattered reads in flight

__global__ void __launch_bounds__(kGatherWarps * 32)
k_gather(int n, int mmax, const AtomS* __restrict__ atoms, const int* __restrict__ nbr_cnt,
         const int* __restrict__ nbr_idx, const unsigned char* __restrict__ rev, const double* __restrict__ pairf,
         const double* __restrict__ e_s, const double* __restrict__ v_s, double* __restrict__ e_out,
         double* __restrict__ f_out, double* __restrict__ var_out, int* __restrict__ flags) {
    constexpr int LPA = 32 / kGatherAPW;  // lanes per atom
    const int lane = threadIdx.x & 31;
    const int sub = lane / LPA, l8 = lane % LPA;
    const int k = (blockIdx.x * kGatherWarps + (threadIdx.x >> 5)) * kGatherAPW + sub;
    const int cnt = k < n ? nbr_cnt[k] : 0;
    double fx = 0.0, fy = 0.0, fz = 0.0;
    for (int s = l8; s < cnt; s += LPA) {  // fixed order per lane, fixed reduction tree below: deterministic
        const size_t own = ((size_t)k * mmax + s) * 3;
        const int j = nbr_idx[(size_t)k * mmax + s];
        const size_t oth = ((size_t)j * mmax + rev[(size_t)k * mmax + s]) * 3;
        fx += pairf[own] - pairf[oth];
        fy += pairf[own + 1] - pairf[oth + 1];
        fz += pairf[own + 2] - pairf[oth + 2];
    }
#pragma unroll
    for (int o = LPA / 2; o > 0; o >>= 1) {
        fx += __shfl_xor_sync(kFull, fx, o);
        fy += __shfl_xor_sync(kFull, fy, o);
        fz += __shfl_xor_sync(kFull, fz, o);
    }
    if (l8 == 0 && k < n) {
        const int i = atoms[k].orig;
        const double e = e_s[k], v = var_out ? v_s[k] : 0.0;
        if (f_out) { f_out[3 * (size_t)i] = fx; f_out[3 * (size_t)i + 1] = fy; f_out[3 * (size_t)i + 2] = fz; }
        if (e_out) e_out[i] = e;
        if (var_out) var_out[i] = v;
        // a blown-up step must not go unnoticed (flare_check -> FLARE_ERR_NONFINITE)
        if (!(isfinite(fx) && isfinite(fy) && isfinite(fz) && isfinite(e) && isfinite(v))) atomicOr(flags, kFlagNonFiniteResult);
    }
}

void run_gather(Launcher& L, const Workspace& ws, int n, int mmax, double* e_out, double* f_out, double* var_out) {
    if (n <= 0) return;
    L.launch(k_gather, dim3((n + kGatherWarps * kGatherAPW - 1) / (kGatherWarps * kGatherAPW)), dim3(kGatherWarps * 32), 0, n, mmax,
             (const AtomS*)ws.atoms, (const int*)ws.nbr_cnt, (const int*)ws.nbr_idx, (const unsigned char*)ws.rev,
             (const double*)ws.pairf, (const double*)ws.e_s, (const double*)ws.v_s, e_out, f_out, var_out, ws.flags);
}

}  // namespace flare
