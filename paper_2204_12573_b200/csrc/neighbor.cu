// neighbor.cu -- step a1: cell-list neighbour build ("all the neighbor atoms within a cutoff
// radius"; R5-R7).  Produces, in cell-sorted atom order, a FULL (symmetric) neighbour
// table nbr_idx[N][mmax] + nbr_cnt[N], the reverse-pair index rev[N][mmax] used by the atomics-free
// force gather, the neighbour-species bitmask, and the grouping of atoms into quadratic-form rows.
// With a skin (the default, R22) the build chain makes a CANDIDATE list with cutoffs r_cut + skin and
// only runs when a device-side gate says an atom has moved skin/2 since the last build; every evaluation
// refreshes the sorted positions and filters the candidates with the exact predicate (k_refresh, k_filter,
// k_rev_from_skin), so the neighbour sets themselves are always exact.
#include "kernels.cuh"

namespace flare {

// ------------------------------------------------------------------ wrap + cell assignment
__global__ void k_cell_assign(Grid g, int n, const double* __restrict__ pos, int* __restrict__ cell_of,
                              int* __restrict__ rank_in_cell, int* __restrict__ cell_cnt, int* __restrict__ flags, const int* __restrict__ gate) {
    if (gate != nullptr && *gate == 0) return;  // skin list still valid: nothing to rebuild
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double p[3] = {pos[3 * i], pos[3 * i + 1], pos[3 * i + 2]};
    int c = 0;
    bool bad = false;
#pragma unroll
    for (int d = 0; d < 3; d++) {
        if (!isfinite(p[d])) { bad = true; p[d] = 0.0; }
        double w = g.pbc[d] ? wrap_coord(p[d], g.L[d]) : p[d];
        int k = (int)floor(w * g.inv_cw[d]);
        k = max(0, min(g.nc[d] - 1, k));
        c += k * g.stride[d];
    }
    if (bad) atomicOr(flags, kFlagNonFinite);
    cell_of[i] = c;
    rank_in_cell[i] = atomicAdd(&cell_cnt[c], 1);
}

// ------------------------------------------------------------------ exclusive scan (3 launches)
constexpr int kScanBlock = 1024;

__global__ void k_scan_partial(int n, const int* __restrict__ in, int* __restrict__ out, int* __restrict__ block_sum, const int* __restrict__ gate) {
    if (gate != nullptr && *gate == 0) return;  // skin list still valid: nothing to rebuild
    __shared__ int warp_tot[32];
    int i = blockIdx.x * kScanBlock + threadIdx.x;
    int v = (i < n) ? in[i] : 0;
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    int x = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int y = __shfl_up_sync(kFull, x, o);
        if (lane >= o) x += y;
    }
    if (lane == 31) warp_tot[w] = x;
    __syncthreads();
    if (w == 0) {
        int t = warp_tot[lane];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int y = __shfl_up_sync(kFull, t, o);
            if (lane >= o) t += y;
        }
        warp_tot[lane] = t;
    }
    __syncthreads();
    int prefix = (w > 0 ? warp_tot[w - 1] : 0) + x - v;  // exclusive within the block
    if (i < n) out[i] = prefix;
    if (threadIdx.x == kScanBlock - 1) block_sum[blockIdx.x] = prefix + v;
}

// single block: exclusive scan of the block sums in place
__global__ void k_scan_sums(int nb, int* __restrict__ block_sum, const int* __restrict__ gate) {
    if (gate != nullptr && *gate == 0) return;  // skin list still valid: nothing to rebuild
    __shared__ int carry_s;
    __shared__ int warp_tot[32];
    if (threadIdx.x == 0) carry_s = 0;
    __syncthreads();
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    for (int base = 0; base < nb; base += kScanBlock) {
        int i = base + threadIdx.x;
        int v = (i < nb) ? block_sum[i] : 0;
        int x = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int y = __shfl_up_sync(kFull, x, o);
            if (lane >= o) x += y;
        }
        if (lane == 31) warp_tot[w] = x;
        __syncthreads();
        if (w == 0) {
            int t = warp_tot[lane];
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                int y = __shfl_up_sync(kFull, t, o);
                if (lane >= o) t += y;
            }
            warp_tot[lane] = t;
        }
        __syncthreads();
        int carry = carry_s;
        int prefix = carry + (w > 0 ? warp_tot[w - 1] : 0) + x - v;
        if (i < nb) block_sum[i] = prefix;
        __syncthreads();
        if (threadIdx.x == kScanBlock - 1) carry_s = prefix + v;
        __syncthreads();
    }
}

__global__ void k_scan_add(int n, int* __restrict__ out, const int* __restrict__ block_sum, const int* __restrict__ gate) {
    if (gate != nullptr && *gate == 0) return;  // skin list still valid: nothing to rebuild
    int i = blockIdx.x * kScanBlock + threadIdx.x;
    if (i < n) out[i] += block_sum[blockIdx.x];
}

// out[n] = out[n-1] + in[n-1]
__global__ void k_scan_total(int n, const int* __restrict__ in, int* __restrict__ out, const int* __restrict__ gate) {
    if (gate != nullptr && *gate == 0) return;  // skin list still valid: nothing to rebuild
    if (threadIdx.x == 0 && blockIdx.x == 0) out[n] = (n > 0) ? out[n - 1] + in[n - 1] : 0;
}

void exclusive_scan(Launcher& L, int n, const int* in, int* out /*[n+1]*/, int* block_sum, const int* gate) {
    int nb = (n + kScanBlock - 1) / kScanBlock;
    if (n > 0) {
        L.launch(k_scan_partial, dim3(nb), dim3(kScanBlock), 0, n, in, out, block_sum, gate);
        L.launch(k_scan_sums, dim3(1), dim3(kScanBlock), 0, nb, block_sum, gate);
        L.launch(k_scan_add, dim3(nb), dim3(kScanBlock), 0, n, out, (const int*)block_sum, gate);
    }
    L.launch(k_scan_total, dim3(1), dim3(32), 0, n, in, out, gate);
}

// ------------------------------------------------------------------ counting sort by cell
__global__ void k_scatter(int n, const int* __restrict__ cell_of, const int* __restrict__ rank_in_cell,
                          const int* __restrict__ cell_start, int* __restrict__ order, const int* __restrict__ gate) {
    if (gate != nullptr && *gate == 0) return;  // skin list still valid: nothing to rebuild
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    order[cell_start[cell_of[i]] + rank_in_cell[i]] = i;
}

// The arrival order of atomicAdd inside a cell is not reproducible: sort each cell's (few) atoms by
// their index in the caller's order so that the whole pipeline is run-to-run deterministic.
__global__ void k_sort_cells(int n_cells, const int* __restrict__ cell_start, int* __restrict__ order, const int* __restrict__ gate) {
    if (gate != nullptr && *gate == 0) return;  // skin list still valid: nothing to rebuild
    int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= n_cells) return;
    int s = cell_start[c], e = cell_start[c + 1];
    for (int a = s + 1; a < e; a++) {
        int v = order[a];
        int b = a - 1;
        while (b >= s && order[b] > v) { order[b + 1] = order[b]; b--; }
        order[b + 1] = v;
    }
}

__global__ void k_gather_atoms(Grid g, int S, int n, const double* __restrict__ pos, const int* __restrict__ types,
                               const int* __restrict__ order, AtomS* __restrict__ atoms, int* __restrict__ flags,
                               const int* __restrict__ gate) {
    if (gate != nullptr && *gate == 0) return;  // skin list still valid: nothing to rebuild
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    int i = order[k];
    AtomS a;
    double p[3] = {pos[3 * i], pos[3 * i + 1], pos[3 * i + 2]};
#pragma unroll
    for (int d = 0; d < 3; d++) {
        if (!isfinite(p[d])) p[d] = 0.0;
        if (g.pbc[d]) p[d] = wrap_coord(p[d], g.L[d]);
    }
    a.x = p[0]; a.y = p[1]; a.z = p[2];
    int t = types[i];
    if ((unsigned)t >= (unsigned)S) { atomicOr(flags, kFlagBadType); t = 0; }  // keeps every table index in bounds
    a.type = t;
    a.orig = i;
    atoms[k] = a;
}

// ------------------------------------------------------------------ neighbour build: warp per atom
__device__ __forceinline__ int fast_ranges(const Grid& g, int cf, int lo_out[2], int hi_out[2]) {
    const int f = g.fast;
    const int nc = g.nc[f];
    if (g.pbc[f]) {
        if (nc <= 3) { lo_out[0] = 0; hi_out[0] = nc - 1; return 1; }  // the whole column, each cell once
        const int lo = cf - 1, hi = cf + 1;
        if (lo < 0) { lo_out[0] = 0; hi_out[0] = hi; lo_out[1] = nc - 1; hi_out[1] = nc - 1; return 2; }
        if (hi >= nc) { lo_out[0] = 0; hi_out[0] = 0; lo_out[1] = lo; hi_out[1] = nc - 1; return 2; }
        lo_out[0] = lo; hi_out[0] = hi;
        return 1;
    }
    lo_out[0] = max(cf - 1, 0);
    hi_out[0] = min(cf + 1, nc - 1);
    return 1;
}

// offsets of a slow dimension: returns count and the (wrapped) cell coordinates
__device__ __forceinline__ int slow_cells(const Grid& g, int d, int c, int out[3]) {
    const int nc = g.nc[d];
    if (g.pbc[d]) {
        if (nc == 1) { out[0] = 0; return 1; }
        if (nc == 2) { out[0] = 0; out[1] = 1; return 2; }
        out[0] = (c + nc - 1) % nc; out[1] = c; out[2] = (c + 1) % nc;
        return 3;
    }
    int k = 0;
    if (c - 1 >= 0) out[k++] = c - 1;
    out[k++] = c;
    if (c + 1 < nc) out[k++] = c + 1;
    return k;
}

constexpr int kNbrWarps = 8;

// One warp per atom.  The (up to 3 x 3 x 2) contiguous runs of candidate atoms -- one per (slow1, slow0)
// cell column and fast-dimension range -- are looked up by the first lanes in parallel, laid end to end by a
// warp scan, and the concatenation is swept 32 candidates at a time, so that every lane tests one candidate
// per sweep whatever the run lengths are (a sweep per run would leave most lanes idle: a run holds ~15 atoms).
__global__ void __launch_bounds__(kNbrWarps * 32)
k_neighbors(Grid g, Basis bs, int n, const AtomS* __restrict__ atoms, const int* __restrict__ cell_start, int mmax,
            int* __restrict__ nbr_cnt, int* __restrict__ nbr_idx, unsigned char* __restrict__ nmask,
            int* __restrict__ flags, const int* __restrict__ gate) {
    if (gate != nullptr && *gate == 0) return;  // skin list still valid: nothing to rebuild
    const int lane = threadIdx.x & 31;
    const int k = blockIdx.x * kNbrWarps + (threadIdx.x >> 5);
    if (k >= n) return;
    const AtomS me = load_atom(atoms + k);
    int c[3];
    c[0] = max(0, min(g.nc[0] - 1, (int)floor(me.x * g.inv_cw[0])));
    c[1] = max(0, min(g.nc[1] - 1, (int)floor(me.y * g.inv_cw[1])));
    c[2] = max(0, min(g.nc[2] - 1, (int)floor(me.z * g.inv_cw[2])));
    int ca[3], cb[3], flo[2], fhi[2];
    const int na = slow_cells(g, g.slow0, c[g.slow0], ca);
    const int nb = slow_cells(g, g.slow1, c[g.slow1], cb);
    const int nf = fast_ranges(g, c[g.fast], flo, fhi);
    // run rr = (ib * na + ia) * nf + r: same visiting order as nested loops over (ib, ia, r)
    const int nr = nb * na * nf;  // <= 18
    int rs = 0, len = 0;
    if (lane < nr) {
        const int r = lane % nf, t = lane / nf;
        const int ia = t % na, ib = t / na;
        const int base = ca[ia] * g.stride[g.slow0] + cb[ib] * g.stride[g.slow1];
        rs = __ldg(cell_start + base + flo[r]);
        len = __ldg(cell_start + base + fhi[r] + 1) - rs;
    }
    int inc = len;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int y = __shfl_up_sync(kFull, inc, o);
        if (lane >= o) inc += y;
    }
    const int total = __shfl_sync(kFull, inc, 31);
    const int exc = inc - len;  // position of the run's first candidate in the concatenation
    int* row = nbr_idx + (size_t)k * mmax;
    int cnt = 0;
    unsigned mask = 0;
    const double* rc2 = bs.rc2 + me.type * bs.S;
    for (int c0 = 0; c0 < total; c0 += 32) {
        const int ci = c0 + lane;
        // last run whose first position is <= ci (empty runs share their successor's position and lose the tie)
        int pos = 0;
#pragma unroll
        for (int st = 16; st > 0; st >>= 1) {
            const int t = pos + st;
            const int v = __shfl_sync(kFull, exc, t & 31);
            if (t < 32 && v <= ci) pos = t;
        }
        const int q = __shfl_sync(kFull, rs, pos) + (ci - __shfl_sync(kFull, exc, pos));
        bool hit = false;
        int tj = 0;
        if (ci < total && q != k) {
            const AtomS o = load_atom(atoms + q);
            double dx, dy, dz;
            displacement(g, me, o, dx, dy, dz);
            tj = o.type;
            hit = dist2_canonical(dx, dy, dz) < rc2[tj];  // strict (R6)
        }
        const unsigned b = __ballot_sync(kFull, hit);
        if (hit) {
            const int slot = cnt + __popc(b & ((1u << lane) - 1u));
            if (slot < mmax) row[slot] = q;
            mask |= 1u << tj;
        }
        cnt += __popc(b);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mask |= __shfl_xor_sync(kFull, mask, o);
    if (lane == 0) {
        if (cnt > mmax) { atomicOr(flags, kFlagNeighborOverflow); cnt = mmax; }
        nbr_cnt[k] = cnt;
        nmask[k] = (unsigned char)mask;
    }
}

// Thread per atom (the default for mmax <= 64).  A CTA takes 128 consecutive cell-sorted atoms; every thread walks the
// (up to 18) candidate runs of its own cell neighbourhood, testing one candidate per iteration.  Threads of a warp sit
// in the same or adjacent cells, so their candidate loads hit the same few 32-byte sectors (L1 broadcast), and the
// per-candidate cost is the ~20 instructions of the canonical distance test instead of a warp-wide sweep with shuffles.
// Hits are staged in shared memory (one padded row per thread) and copied out as coalesced rows.
constexpr int kNbrThreads = 128;

__global__ void __launch_bounds__(kNbrThreads)
k_neighbors_tpa(Grid g, Basis bs, int n, const AtomS* __restrict__ atoms, const int* __restrict__ cell_start, int mmax,
                int* __restrict__ nbr_cnt, int* __restrict__ nbr_idx, unsigned char* __restrict__ nmask,
                int* __restrict__ flags, const int* __restrict__ gate) {
    if (gate != nullptr && *gate == 0) return;  // skin list still valid: nothing to rebuild
    extern __shared__ int stage[];  // [kNbrThreads][mmax | 1]
    const int ST = mmax | 1;
    const int k = blockIdx.x * kNbrThreads + threadIdx.x;
    int cnt = 0;
    unsigned mask = 0;
    if (k < n) {
        const AtomS me = load_atom(atoms + k);
        int c[3];
        c[0] = max(0, min(g.nc[0] - 1, (int)floor(me.x * g.inv_cw[0])));
        c[1] = max(0, min(g.nc[1] - 1, (int)floor(me.y * g.inv_cw[1])));
        c[2] = max(0, min(g.nc[2] - 1, (int)floor(me.z * g.inv_cw[2])));
        int ca[3], cb[3], flo[2], fhi[2];
        const int na = slow_cells(g, g.slow0, c[g.slow0], ca);
        const int nb = slow_cells(g, g.slow1, c[g.slow1], cb);
        const int nf = fast_ranges(g, c[g.fast], flo, fhi);
        const double* rc2 = bs.rc2 + me.type * bs.S;
        int* row = stage + threadIdx.x * ST;
        for (int ib = 0; ib < nb; ib++)
            for (int ia = 0; ia < na; ia++) {
                const int base = ca[ia] * g.stride[g.slow0] + cb[ib] * g.stride[g.slow1];
                for (int r = 0; r < nf; r++) {
                    const int qs = __ldg(cell_start + base + flo[r]);
                    const int qe = __ldg(cell_start + base + fhi[r] + 1);
                    for (int q = qs; q < qe; q++) {
                        if (q == k) continue;
                        const AtomS o = load_atom(atoms + q);
                        double dx, dy, dz;
                        displacement(g, me, o, dx, dy, dz);
                        if (dist2_canonical(dx, dy, dz) < rc2[o.type]) {  // strict (R6)
                            if (cnt < mmax) row[cnt] = q;
                            cnt++;
                            mask |= 1u << o.type;
                        }
                    }
                }
            }
        if (cnt > mmax) { atomicOr(flags, kFlagNeighborOverflow); cnt = mmax; }
        nbr_cnt[k] = cnt;
        nmask[k] = (unsigned char)mask;
    }
    // coalesced copy-out: each warp writes the rows of its own 32 threads, one row at a time
    __syncwarp();
    const int lane = threadIdx.x & 31, w0 = threadIdx.x & ~31;
    for (int t = 0; t < 32; t++) {
        const int ct = __shfl_sync(kFull, cnt, t);
        const int kt = blockIdx.x * kNbrThreads + w0 + t;
        const int* src = stage + (w0 + t) * ST;
        for (int s = lane; s < ct; s += 32) nbr_idx[(size_t)kt * mmax + s] = src[s];
    }
}

// rev[k][s] = slot of k in the row of j = nbr_idx[k][s]  (exists because cutoffs are symmetric, R5).
// Lane s holds neighbour s and its row length; the rows of four neighbours are fetched together (one
// coalesced 128-byte read each) before any of them is searched, and the found slots are written back as
// one coalesced byte store per 32 neighbours.
__global__ void __launch_bounds__(kNbrWarps * 32)
k_reverse_index(int n, int mmax, const int* __restrict__ nbr_cnt, const int* __restrict__ nbr_idx,
                unsigned char* __restrict__ rev, const int* __restrict__ gate) {
    if (gate != nullptr && *gate == 0) return;  // skin list still valid: nothing to rebuild
    const int lane = threadIdx.x & 31;
    // grid-stride over atoms: a fixed, small grid, so that the gated (skipped) launch costs next to nothing
    for (int k = blockIdx.x * kNbrWarps + (threadIdx.x >> 5); k < n; k += gridDim.x * kNbrWarps) {
        const int cnt = nbr_cnt[k];
        for (int base = 0; base < cnt; base += 32) {
            const int s = base + lane;
            const int nact = min(32, cnt - base);
            int j = 0, cj = 0;
            if (s < cnt) { j = nbr_idx[(size_t)k * mmax + s]; cj = nbr_cnt[j]; }
            int mine = 0;
            for (int t0 = 0; t0 < nact; t0 += 4) {
                int jj[4], cc[4], v[4];
#pragma unroll
                for (int u = 0; u < 4; u++) {
                    jj[u] = __shfl_sync(kFull, j, (t0 + u) & 31);
                    cc[u] = __shfl_sync(kFull, cj, (t0 + u) & 31);  // 0 beyond nact: nothing is read
                    v[u] = (lane < cc[u]) ? nbr_idx[(size_t)jj[u] * mmax + lane] : -1;
                }
#pragma unroll
                for (int u = 0; u < 4; u++) {
                    unsigned m = __ballot_sync(kFull, v[u] == k);
                    int found = m ? __ffs(m) - 1 : 0;
                    for (int b = 32; !m && b < cc[u]; b += 32) {  // rows longer than a warp
                        const int t = b + lane;
                        m = __ballot_sync(kFull, (t < cc[u]) && (nbr_idx[(size_t)jj[u] * mmax + t] == k));
                        if (m) found = b + __ffs(m) - 1;
                    }
                    if (lane == t0 + u) mine = found;
                }
            }
            if (s < cnt) rev[(size_t)k * mmax + s] = (unsigned char)mine;
        }
    }
}

// ------------------------------------------------------------------ skin list (R12: "a skin list filtered by the exact
// predicate is allowed, sets must still be exact").  Between rebuilds the cell-sorted order and a candidate list built
// with the cutoff max r_cut + skin are kept; every evaluation refreshes the sorted positions, checks the per-species
// displacements since the build against the budget of every species pair (else the gate is raised and the whole build
// chain above runs again), and filters the candidates with the exact canonical predicate.  The reverse-pair index of the
// filtered list follows from the candidate list's own reverse index and the per-atom hit masks, without any search.

// sorted positions <- current positions (in the order of the last build); per-species maximum displacement since the
// build (as the bits of a float rounded up: non-negative floats order like their bit patterns) -> dmax[S]
__global__ void k_refresh(Grid g, int S, int n, const double* __restrict__ pos, const int* __restrict__ types,
                          const int* __restrict__ order, const AtomS* __restrict__ ref, AtomS* __restrict__ atoms,
                          int* __restrict__ gate, int* __restrict__ dmax, int* __restrict__ flags,
                          const double* __restrict__ dom_ref, double dom_trigger2, double dom_limit2,
                          int* __restrict__ dom_need) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    int my_type = -1;
    int bits = 0;
    if (k < n) {
        const int i = order[k];
        double p[3] = {pos[3 * (size_t)i], pos[3 * (size_t)i + 1], pos[3 * (size_t)i + 2]};
        bool bad = false;
#pragma unroll
        for (int d = 0; d < 3; d++) {
            if (!isfinite(p[d])) { bad = true; p[d] = 0.0; }
            if (g.pbc[d]) p[d] = wrap_coord(p[d], g.L[d]);
        }
        if (dom_ref) {
            // domain decomposition (domain.cu): the ghost shell was chosen for the positions of the last domain rebuild
            // and tolerates a displacement of dom_trigger per atom, whatever the candidate list did in between
            double d2 = 0.0;
#pragma unroll
            for (int d = 0; d < 3; d++) {
                double r = dom_ref[3 * (size_t)i + d];
                if (g.pbc[d]) r = wrap_coord(r, g.L[d]);
                const double dd = min_image(p[d] - r, g.L[d], g.half[d], g.pbc[d]);
                d2 += dd * dd;
            }
            if (!(d2 < dom_trigger2)) *dom_need = 1;  // benign race: every writer stores 1
            // the rebuild asked for above arrives a few steps later (the signal is all-reduced and read with a lag):
            // past dom_limit the shell no longer holds every ghost an owned atom's force needs -- an error, not a signal
            if (!(d2 < dom_limit2)) atomicOr(flags, kFlagHaloExceeded);
        }
        AtomS a;
        a.x = p[0]; a.y = p[1]; a.z = p[2];
        int t = types[i];
        if ((unsigned)t >= (unsigned)S) { atomicOr(flags, kFlagBadType); t = 0; }
        a.type = t;
        a.orig = i;
        atoms[k] = a;
        const AtomS r = load_atom(ref + k);
        double dx, dy, dz;
        displacement(g, r, a, dx, dy, dz);
        const double d2 = dx * dx + dy * dy + dz * dz;
        if (bad) atomicOr(flags, kFlagNonFinite);
        if (bad || !(d2 < 1e30) || r.type != a.type) *gate = 1;  // benign race: every writer stores 1
        my_type = a.type;
        bits = __float_as_int(__double2float_ru(sqrt(d2)));
    }
    // one atomic per (warp, species present in the warp)
    for (int s = 0; s < S; s++) {
        int m = (my_type == s) ? bits : 0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) m = max(m, __shfl_xor_sync(kFull, m, o));
        if ((threadIdx.x & 31) == 0 && m > 0) atomicMax(dmax + s, m);
    }
}

// A pair (a, b) of the candidate list (cutoff rc_max + skin for every pair) stays complete while
// d_a + d_b < (rc_max + skin) - r_cut[a][b]: the pairs with the largest cutoff have `skin` to spend, pairs with a
// shorter cutoff (every pair with an H in the H2/Pt workloads) much more, so the fast light atoms do not force
// rebuilds.  The threshold is taken a hair low so that the triangle inequality holds with rounding to spare.
// In a captured step (CUDA graph, small systems) the decision also drives the IF node that holds the rebuild chain.
__global__ void k_gate_decide(Basis bs, double reach, const int* __restrict__ dmax, int* __restrict__ gate,
                              cudaGraphConditionalHandle cond, int use_cond) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    int need = *gate;  // k_refresh raises it for a non-finite position or a changed species
    for (int a = 0; a < bs.S; a++)
        for (int b = a; b < bs.S; b++) {
            const double da = __int_as_float(dmax[a]), db = __int_as_float(dmax[b]);
            if (!(da + db < 0.9998 * (reach - bs.rc[a * bs.S + b]))) need = 1;
        }
    if (need) *gate = 1;
    if (use_cond) cudaGraphSetConditional(cond, need ? 1u : 0u);
}

__global__ void k_copy_ref(int n, const AtomS* __restrict__ atoms, AtomS* __restrict__ ref, const int* __restrict__ gate,
                           int* __restrict__ n_rebuilds) {
    if (gate != nullptr && *gate == 0) return;
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k < n) ref[k] = atoms[k];
    if (k == 0) *n_rebuilds += 1;  // statistics (FLARE_OPT_SKIN_REBUILDS)
}

// A warp takes kFilterAtoms consecutive atoms, 8 lanes each: a lane tests candidates l8, l8 + 8, ... of its atom's skin row
// with the exact predicate, four at a time, their index and atom loads issued before the first test (the kernel is bound
// by the latency of the scattered 32-byte atom reads: with ~22 candidates per row, 8 lanes per atom keep the lanes full
// and three to four reads per lane in flight); hits are compacted into nbr_idx, in candidate order, by ballot.
constexpr int kFilterAtoms = 4;  // atoms per warp: 8 lanes each

__global__ void __launch_bounds__(kNbrWarps * 32)
k_filter(Grid g, Basis bs, int n, int mmax, int smax, const AtomS* __restrict__ atoms, const int* __restrict__ skin_cnt,
         const int* __restrict__ skin_idx, int* __restrict__ nbr_cnt, int* __restrict__ nbr_idx,
         unsigned char* __restrict__ nmask, unsigned long long* __restrict__ hitmask, int* __restrict__ flags) {
    constexpr int LPA = 32 / kFilterAtoms;  // lanes per atom
    constexpr int UN = 4;                   // candidates per lane whose loads fly together (UN * LPA = 32 per chunk)
    const int lane = threadIdx.x & 31;
    const int sub = lane / LPA, l8 = lane % LPA;
    const int k = (blockIdx.x * kNbrWarps + (threadIdx.x >> 5)) * kFilterAtoms + sub;
    const bool live = k < n;
    const int sc = live ? skin_cnt[k] : 0;
    const AtomS me = load_atom(atoms + (live ? k : 0));
    const unsigned grp = ((1u << LPA) - 1u) << (sub * LPA);  // ballot bits of this atom's lanes
    int cnt = 0;
    unsigned mask = 0;
    unsigned long long hm = 0;
    int scmax = sc;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) scmax = max(scmax, __shfl_xor_sync(kFull, scmax, o));
    for (int base = 0; base < scmax; base += UN * LPA) {  // at most 2 chunks (rows hold <= 64 candidates)
        int j[UN];
        AtomS o[UN];
#pragma unroll
        for (int u = 0; u < UN; u++) {
            const int s = base + u * LPA + l8;
            j[u] = (s < sc) ? skin_idx[(size_t)k * smax + s] : 0;
        }
#pragma unroll
        for (int u = 0; u < UN; u++) o[u] = load_atom(atoms + j[u]);
#pragma unroll
        for (int u = 0; u < UN; u++) {  // candidate order s = base + u LPA + l8: ascending in (u, lane), as the list expects
            const int s = base + u * LPA + l8;
            double dx, dy, dz;
            displacement(g, me, o[u], dx, dy, dz);
            const bool hit = (s < sc) && dist2_canonical(dx, dy, dz) < bs.rc2[me.type * bs.S + o[u].type];  // strict (R6)
            const unsigned b = __ballot_sync(kFull, hit) & grp;
            if (hit) {
                const int slot = cnt + __popc(b & ((1u << lane) - 1u));
                if (slot < mmax) nbr_idx[(size_t)k * mmax + slot] = j[u];
                mask |= 1u << o[u].type;
                hm |= 1ull << s;
            }
            cnt += __popc(b);
        }
    }
#pragma unroll
    for (int o = LPA / 2; o > 0; o >>= 1) {
        mask |= __shfl_xor_sync(kFull, mask, o);
        hm |= __shfl_xor_sync(kFull, hm, o);
    }
    if (l8 == 0 && live) {
        if (cnt > mmax) { atomicOr(flags, kFlagNeighborOverflow); cnt = mmax; }
        nbr_cnt[k] = cnt;
        nmask[k] = (unsigned char)mask;
        hitmask[k] = hm;
    }
}

constexpr int kRevAtoms = 4;  // atoms per warp pass in k_rev_from_skin: their scattered hit-mask reads fly together

// rev of the filtered list: the hit (k, s) sits in row j at the number of j's hits before k's candidate slot there
__global__ void __launch_bounds__(kNbrWarps * 32)
k_rev_from_skin(int n, int mmax, int smax, const int* __restrict__ skin_cnt, const int* __restrict__ skin_idx,
                const unsigned char* __restrict__ skin_rev, const unsigned long long* __restrict__ hitmask,
                unsigned char* __restrict__ rev) {
    const int lane = threadIdx.x & 31;
    const int k0 = (blockIdx.x * kNbrWarps + (threadIdx.x >> 5)) * kRevAtoms;
    if (k0 >= n) return;
    int sc[kRevAtoms];
    unsigned long long hm[kRevAtoms];
    int scmax = 0;
#pragma unroll
    for (int a = 0; a < kRevAtoms; a++) {
        const bool in = k0 + a < n;
        sc[a] = in ? skin_cnt[k0 + a] : 0;
        hm[a] = in ? hitmask[k0 + a] : 0ull;
        scmax = max(scmax, sc[a]);
    }
    for (int base = 0; base < scmax; base += 32) {
        const int s = base + lane;
        bool on[kRevAtoms];
        int t[kRevAtoms];
        unsigned long long hj[kRevAtoms];
#pragma unroll
        for (int a = 0; a < kRevAtoms; a++) {
            on[a] = s < sc[a] && ((hm[a] >> s) & 1ull);
            const size_t q = (size_t)(k0 + a) * smax + s;
            const int j = on[a] ? skin_idx[q] : 0;
            t[a] = on[a] ? skin_rev[q] : 0;  // candidate slot of k in row j
            hj[a] = hitmask[j];
        }
#pragma unroll
        for (int a = 0; a < kRevAtoms; a++) {
            if (on[a]) {
                const int slot = __popcll(hm[a] & ((1ull << s) - 1ull));
                if (slot < mmax)
                    rev[(size_t)(k0 + a) * mmax + slot] = (unsigned char)__popcll(hj[a] & ((1ull << t[a]) - 1ull));
            }
        }
    }
}

// ------------------------------------------------------------------ grouping into quadratic-form rows
// Group of an atom: dense mode -> its species; sparse mode -> (species, neighbour-species mask).
__device__ __forceinline__ int group_of(int type, unsigned mask, int S, int sparse) {
    return sparse ? type * (1 << S) + (int)mask : type;
}

constexpr int kGroupBlock = 1024;

__global__ void __launch_bounds__(kGroupBlock)
k_group_hist(int n, int S, int sparse, int n_groups, const AtomS* __restrict__ atoms,
             const unsigned char* __restrict__ nmask, int* __restrict__ hist /*[n_blocks][n_groups]*/) {
    __shared__ int h[kMaxGroups];
    for (int t = threadIdx.x; t < n_groups; t += blockDim.x) h[t] = 0;
    __syncthreads();
    int k = blockIdx.x * kGroupBlock + threadIdx.x;
    if (k < n) atomicAdd(&h[group_of(atoms[k].type, nmask[k], S, sparse)], 1);
    __syncthreads();
    for (int t = threadIdx.x; t < n_groups; t += blockDim.x) hist[(size_t)blockIdx.x * n_groups + t] = h[t];
}

// one warp per group scans that group's per-block counts (exclusive, in place); then thread 0 lays the groups
// out one after another
__global__ void __launch_bounds__(32 * 32)
k_group_scan(int n_blocks, int n_groups, int* __restrict__ hist, int* __restrict__ group_start) {
    __shared__ int tot[kMaxGroups + 1];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    for (int gidx = w; gidx < n_groups; gidx += 32) {
        int run = 0;
        for (int b0 = 0; b0 < n_blocks; b0 += 32) {
            const int b = b0 + lane;
            const int v = (b < n_blocks) ? hist[(size_t)b * n_groups + gidx] : 0;
            int x = v;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int y = __shfl_up_sync(kFull, x, o);
                if (lane >= o) x += y;
            }
            if (b < n_blocks) hist[(size_t)b * n_groups + gidx] = run + x - v;
            run += __shfl_sync(kFull, x, 31);
        }
        if (lane == 0) tot[gidx] = run;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        int run = 0;
        for (int t = 0; t < n_groups; t++) { group_start[t] = run; run += tot[t]; }
        group_start[n_groups] = run;
    }
}

__global__ void __launch_bounds__(kGroupBlock)
k_group_assign(int n, int S, int sparse, int n_groups, const AtomS* __restrict__ atoms,
               const unsigned char* __restrict__ nmask, const int* __restrict__ hist,
               const int* __restrict__ group_start, int* __restrict__ row_of, int* __restrict__ atom_of_row,
               unsigned char* __restrict__ gid_out) {
    __shared__ int wcnt[32][kMaxGroups];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    for (int t = threadIdx.x; t < 32 * kMaxGroups; t += blockDim.x) (&wcnt[0][0])[t] = 0;
    __syncthreads();
    const int k = blockIdx.x * kGroupBlock + threadIdx.x;
    const int gid = (k < n) ? group_of(atoms[k].type, nmask[k], S, sparse) : -1;
    const unsigned peers = __match_any_sync(kFull, gid);
    const int rank = __popc(peers & ((1u << lane) - 1u));
    if (gid >= 0 && rank == 0) wcnt[w][gid] = __popc(peers);
    __syncthreads();
    if (gid >= 0) {
        int before = 0;
        for (int ww = 0; ww < w; ww++) before += wcnt[ww][gid];
        const int row = group_start[gid] + hist[(size_t)blockIdx.x * n_groups + gid] + before + rank;
        row_of[k] = row;
        atom_of_row[row] = k;
        gid_out[k] = (unsigned char)gid;
    }
}

// n <= kGroupBlock: histogram, scan and assignment in one block and one launch (a small step is bound by the latency of
// its chain of tiny kernels); same row order as the three-kernel version
__global__ void __launch_bounds__(kGroupBlock)
k_group_small(int n, int S, int sparse, int n_groups, const AtomS* __restrict__ atoms,
              const unsigned char* __restrict__ nmask, int* __restrict__ group_start, int* __restrict__ row_of,
              int* __restrict__ atom_of_row, unsigned char* __restrict__ gid_out) {
    __shared__ int wcnt[32][kMaxGroups];
    __shared__ int start[kMaxGroups + 1];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    for (int t = threadIdx.x; t < 32 * kMaxGroups; t += blockDim.x) (&wcnt[0][0])[t] = 0;
    __syncthreads();
    const int k = threadIdx.x;
    const int gid = (k < n) ? group_of(atoms[k].type, nmask[k], S, sparse) : -1;
    const unsigned peers = __match_any_sync(kFull, gid);
    const int rank = __popc(peers & ((1u << lane) - 1u));
    if (gid >= 0 && rank == 0) wcnt[w][gid] = __popc(peers);
    __syncthreads();
    if (threadIdx.x < n_groups) {  // total of each group ...
        int tot = 0;
        for (int ww = 0; ww < 32; ww++) tot += wcnt[ww][threadIdx.x];
        start[threadIdx.x + 1] = tot;
    }
    __syncthreads();
    if (threadIdx.x == 0) {  // ... laid out one after another
        start[0] = 0;
        for (int gq = 0; gq < n_groups; gq++) start[gq + 1] += start[gq];
        for (int gq = 0; gq <= n_groups; gq++) group_start[gq] = start[gq];
    }
    __syncthreads();
    if (gid >= 0) {
        int before = 0;
        for (int ww = 0; ww < w; ww++) before += wcnt[ww][gid];
        const int row = start[gid] + before + rank;
        row_of[k] = row;
        atom_of_row[row] = k;
        gid_out[k] = (unsigned char)gid;
    }
}

// ------------------------------------------------------------------ host-side driver of a1
void build_neighbors(Launcher& L, const Grid& g, const Basis& bs, const Workspace& ws, int n, const double* pos,
                     const int* types, int mmax, int sparse, int n_groups, double skin, bool list_valid,
                     double dom_trigger, double dom_limit) {
    if (n == 0) return;
    const int tb = 256;
    const bool use_skin = skin > 0.0;
    const int* gate = nullptr;
    int* nbr_cnt = ws.nbr_cnt;
    int* nbr_idx = ws.nbr_idx;
    unsigned char* rev = ws.rev;
    Basis bsb = bs;  // cutoffs of the list that is BUILT (r_cut + skin in skin mode)
    int bmax = mmax;  // its row stride
    if (use_skin) {
        bmax = kSkinStride;
        gate = ws.skin_gate;
        nbr_cnt = ws.skin_cnt; nbr_idx = ws.skin_idx; rev = ws.skin_rev;
        double rcmax = 0.0;
        for (int i = 0; i < bs.S * bs.S; i++) rcmax = bs.rc[i] > rcmax ? bs.rc[i] : rcmax;
        const double reach = rcmax + skin;  // one candidate cutoff for every species pair
        for (int i = 0; i < bs.S * bs.S; i++) bsb.rc2[i] = reach * reach;
        L.memset(ws.skin_gate, list_valid ? 0 : 1, sizeof(int));  // bytes of 0x01: non-zero = rebuild; [1] counts rebuilds
        if (list_valid) {
            L.memset(ws.skin_gate + 4, 0, sizeof(int) * kMaxSpecies);  // per-species maximum displacement
            L.launch(k_refresh, dim3((n + tb - 1) / tb), dim3(tb), 0, g, bs.S, n, pos, types, (const int*)ws.order,
                     (const AtomS*)ws.ref, ws.atoms, ws.skin_gate, ws.skin_gate + 4, ws.flags,
                     dom_trigger > 0.0 || dom_limit > 0.0 ? (const double*)ws.dom_ref : (const double*)nullptr,
                     dom_trigger > 0.0 ? dom_trigger * dom_trigger : HUGE_VAL,
                     dom_limit > 0.0 ? dom_limit * dom_limit : HUGE_VAL, ws.dom + kDomNeed);
            // captured step: the rebuild chain below becomes the body of an IF node that k_gate_decide switches on,
            // so a step that keeps its list pays for none of the chain's (otherwise empty) launches
            const bool as_if = L.capturing;
            const cudaGraphConditionalHandle h = as_if ? L.cond_handle() : 0;
            L.launch(k_gate_decide, dim3(1), dim3(32), 0, bs, reach, (const int*)(ws.skin_gate + 4), ws.skin_gate, h,
                     as_if ? 1 : 0);
            if (as_if) { L.begin_if(h); gate = nullptr; }
        }
    }
    L.memset(ws.cell_cnt, 0, sizeof(int) * (size_t)g.n_cells);
    L.launch(k_cell_assign, dim3((n + tb - 1) / tb), dim3(tb), 0, g, n, pos, ws.cell_of, ws.rank_in_cell, ws.cell_cnt,
             ws.flags, gate);
    exclusive_scan(L, g.n_cells, ws.cell_cnt, ws.cell_start, ws.scan_tmp, gate);
    L.launch(k_scatter, dim3((n + tb - 1) / tb), dim3(tb), 0, n, (const int*)ws.cell_of, (const int*)ws.rank_in_cell,
             (const int*)ws.cell_start, ws.order, gate);
    L.launch(k_sort_cells, dim3((g.n_cells + tb - 1) / tb), dim3(tb), 0, g.n_cells, (const int*)ws.cell_start, ws.order,
             gate);
    L.launch(k_gather_atoms, dim3((n + tb - 1) / tb), dim3(tb), 0, g, bs.S, n, pos, types, (const int*)ws.order, ws.atoms,
             ws.flags, gate);
    const int nwb = (n + kNbrWarps - 1) / kNbrWarps;
    if (bmax <= 64) {
        const size_t stage = sizeof(int) * kNbrThreads * (size_t)(bmax | 1);
        L.launch(k_neighbors_tpa, dim3((n + kNbrThreads - 1) / kNbrThreads), dim3(kNbrThreads), stage, g, bsb, n,
                 (const AtomS*)ws.atoms, (const int*)ws.cell_start, bmax, nbr_cnt, nbr_idx, ws.nmask, ws.flags, gate);
    } else {
        L.launch(k_neighbors, dim3(nwb), dim3(kNbrWarps * 32), 0, g, bsb, n, (const AtomS*)ws.atoms,
                 (const int*)ws.cell_start, bmax, nbr_cnt, nbr_idx, ws.nmask, ws.flags, gate);
    }
    L.launch(k_reverse_index, dim3(nwb < 148 * 32 ? nwb : 148 * 32), dim3(kNbrWarps * 32), 0, n, bmax, (const int*)nbr_cnt, (const int*)nbr_idx, rev,
             gate);
    if (use_skin) {
        L.launch(k_copy_ref, dim3((n + tb - 1) / tb), dim3(tb), 0, n, (const AtomS*)ws.atoms, ws.ref, gate, ws.skin_gate + 1);
        L.end_if();  // no-op unless the chain was captured as an IF body
        const int nfb = (n + kNbrWarps * kFilterAtoms - 1) / (kNbrWarps * kFilterAtoms);
        L.launch(k_filter, dim3(nfb), dim3(kNbrWarps * 32), 0, g, bs, n, mmax, bmax, (const AtomS*)ws.atoms,
                 (const int*)ws.skin_cnt, (const int*)ws.skin_idx, ws.nbr_cnt, ws.nbr_idx, ws.nmask, ws.hitmask, ws.flags);
        const int nrb = (n + kNbrWarps * kRevAtoms - 1) / (kNbrWarps * kRevAtoms);
        L.launch(k_rev_from_skin, dim3(nrb), dim3(kNbrWarps * 32), 0, n, mmax, bmax, (const int*)ws.skin_cnt,
                 (const int*)ws.skin_idx, (const unsigned char*)ws.skin_rev, (const unsigned long long*)ws.hitmask, ws.rev);
    }
    const int ngb = (n + kGroupBlock - 1) / kGroupBlock;
    if (ngb == 1) {
        L.launch(k_group_small, dim3(1), dim3(kGroupBlock), 0, n, bs.S, sparse, n_groups, (const AtomS*)ws.atoms,
                 (const unsigned char*)ws.nmask, ws.group_start, ws.row_of, ws.atom_of_row, ws.gid);
        return;
    }
    L.launch(k_group_hist, dim3(ngb), dim3(kGroupBlock), 0, n, bs.S, sparse, n_groups, (const AtomS*)ws.atoms,
             (const unsigned char*)ws.nmask, ws.group_hist);
    L.launch(k_group_scan, dim3(1), dim3(32 * 32), 0, ngb, n_groups, ws.group_hist, ws.group_start);
    L.launch(k_group_assign, dim3(ngb), dim3(kGroupBlock), 0, n, bs.S, sparse, n_groups, (const AtomS*)ws.atoms,
             (const unsigned char*)ws.nmask, (const int*)ws.group_hist, (const int*)ws.group_start, ws.row_of,
             ws.atom_of_row, ws.gid);
}

}  // namespace flare
