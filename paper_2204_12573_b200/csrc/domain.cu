// domain.cu -- device data plane of the multi-GPU domain decomposition ("MD runs
// entirely on GPUs with zero CPU-GPU data transfer except for I/O", "near-two-dimensional").
//
// One process per GPU owns the atoms of one rectangle of the (x, y) plane and evaluates them together with ghost
// copies of every atom within the halo width of the rectangle.  The state arrays of the bound context hold
//     [ owned atoms 0 .. n_owned ) [ ghosts of the x phase ) [ ghosts of the y phase )
// in a LOCAL frame (decomposed dimensions open, rectangle at [halo, halo + w)), so a neighbour's frame differs from
// mine by +- w along the axis and periodic images need no special case.  This file holds the kernels that
//   * select, in index order (stable, so that results do not depend on thread scheduling), the atoms that leave
//     through a face (migration) or lie within the halo width of a face (border), and pack them into messages;
//   * compact the atoms that stay and append arrivals / ghosts;
//   * per MD step, gather (x + shift, v, F) of the fixed send lists into messages and scatter received rows into the
//     fixed ghost slots: between two rebuilds membership, order and counts do not change, so the candidate
//     neighbour list of the context survives and no message size has to be communicated.
// Messages are plain double arrays: [0] = row count, rows start at double 8; a full row is
// (x, y, z, vx, vy, vz, fx, fy, fz, type, tag) = 11 doubles, a forward row (x, y, z, vx, vy, vz, fx, fy, fz) = 9.
// All counts live in device memory (Workspace::dom): no kernel here needs the host to know a size.
#include <algorithm>

#include "kernels.cuh"

namespace flare {

constexpr int kDomBlock = 1024;

// bit 0: the coordinate lies in [lo_a, lo_b) (-> "lo" list), bit 1: in [hi_a, hi_b) (-> "hi" list)
__device__ __forceinline__ int dom_code(double x, const DomSel& s) {
    return ((x >= s.lo_a && x < s.lo_b) ? 1 : 0) | ((x >= s.hi_a && x < s.hi_b) ? 2 : 0);
}

// per block of kDomBlock atoms: members of the lo list, of the hi list, and atoms in neither ("stay")
__global__ void __launch_bounds__(kDomBlock)
k_dom_count(DomSel s, const int* __restrict__ dom, const double* __restrict__ x, int* __restrict__ blk) {
    const int n = dom[s.n_from];
    const int i = blockIdx.x * kDomBlock + threadIdx.x;
    const int code = (i < n) ? dom_code(x[3 * (size_t)i + s.axis], s) : -1;
    const int c0 = __syncthreads_count(code >= 0 && (code & 1));
    const int c1 = __syncthreads_count(code >= 0 && (code & 2));
    const int c2 = __syncthreads_count(code == 0);
    if (threadIdx.x == 0) {
        const int nb = gridDim.x;
        blk[blockIdx.x] = c0; blk[nb + blockIdx.x] = c1; blk[2 * nb + blockIdx.x] = c2;
    }
}

// exclusive scan of the three rows of block counts (one block; nb is a few thousand at most); totals -> dom[kDomTot..]
__global__ void __launch_bounds__(1024) k_dom_scan(int nb, int* __restrict__ blk, int* __restrict__ dom) {
    __shared__ int wsum[32];
    __shared__ int carry;
    for (int row = 0; row < 3; row++) {
        if (threadIdx.x == 0) carry = 0;
        __syncthreads();
        for (int base = 0; base < nb; base += 1024) {
            const int i = base + threadIdx.x;
            const int v = (i < nb) ? blk[row * nb + i] : 0;
            int inc = v;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int t = __shfl_up_sync(kFull, inc, o);
                if ((threadIdx.x & 31) >= o) inc += t;
            }
            if ((threadIdx.x & 31) == 31) wsum[threadIdx.x >> 5] = inc;
            __syncthreads();
            if (threadIdx.x < 32) {
                int w = wsum[threadIdx.x];
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const int t = __shfl_up_sync(kFull, w, o);
                    if (threadIdx.x >= o) w += t;
                }
                wsum[threadIdx.x] = w;  // inclusive over warps
            }
            __syncthreads();
            const int before = carry + ((threadIdx.x >> 5) ? wsum[(threadIdx.x >> 5) - 1] : 0) + inc - v;
            if (i < nb) blk[row * nb + i] = before;
            __syncthreads();
            if (threadIdx.x == 1023) carry = before + v;
            __syncthreads();
        }
        if (threadIdx.x == 0) dom[kDomTot + row] = carry;
        __syncthreads();
    }
}

// ordered write of the three index lists (any may be null); entries beyond `cap` (`cap_stay`) are dropped and flagged
__global__ void __launch_bounds__(kDomBlock)
k_dom_write(DomSel s, const int* __restrict__ dom, const double* __restrict__ x, const int* __restrict__ blk,
            int* __restrict__ list_lo, int* __restrict__ list_hi, int* __restrict__ list_stay, int cap, int cap_stay,
            int* __restrict__ flags) {
    __shared__ int wcnt[3][32];
    const int n = dom[s.n_from];
    const int i = blockIdx.x * kDomBlock + threadIdx.x;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int code = (i < n) ? dom_code(x[3 * (size_t)i + s.axis], s) : -1;
    const bool in[3] = {code >= 0 && (code & 1), code >= 0 && (code & 2), code == 0};
    unsigned bal[3];
#pragma unroll
    for (int r = 0; r < 3; r++) {
        bal[r] = __ballot_sync(kFull, in[r]);
        if (lane == 0) wcnt[r][warp] = __popc(bal[r]);
    }
    __syncthreads();
    if (warp < 3) {  // exclusive scan over the 32 warps of row `warp`
        const int v = wcnt[warp][lane];
        int inc = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(kFull, inc, o);
            if (lane >= o) inc += t;
        }
        wcnt[warp][lane] = inc - v;
    }
    __syncthreads();
    int* const lists[3] = {list_lo, list_hi, list_stay};
    const int nb = gridDim.x;
#pragma unroll
    for (int r = 0; r < 3; r++) {
        if (in[r] && lists[r]) {
            const int pos = blk[r * nb + blockIdx.x] + wcnt[r][warp] + __popc(bal[r] & ((1u << lane) - 1u));
            if (pos < (r == 2 ? cap_stay : cap)) lists[r][pos] = i;
            else atomicOr(flags, kFlagDomainOverflow);
        }
    }
}

// send counts of the selection -> dom[slot_lo], dom[slot_hi] (clipped to the list capacity)
__global__ void k_dom_commit_lists(int* __restrict__ dom, int slot_lo, int slot_hi, int cap) {
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        dom[slot_lo] = min(dom[kDomTot + 0], cap);
        dom[slot_hi] = min(dom[kDomTot + 1], cap);
    }
}

// full rows of a list -> message (count in the header; rows beyond the message capacity are dropped and flagged)
__global__ void k_dom_pack_full(const int* __restrict__ list, const int* __restrict__ dom, int cnt_slot, double sx,
                                double sy, double sz, const double* __restrict__ x, const double* __restrict__ v,
                                const double* __restrict__ f, const int* __restrict__ types,
                                const long long* __restrict__ tag, int with_force, double* __restrict__ msg,
                                int cap_rows, int* __restrict__ flags) {
    int cnt = dom[cnt_slot];
    if (cnt > cap_rows) {
        cnt = cap_rows;
        if (blockIdx.x == 0 && threadIdx.x == 0) atomicOr(flags, kFlagDomainOverflow);
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) msg[0] = (double)cnt;
    for (int r = blockIdx.x * blockDim.x + threadIdx.x; r < cnt; r += gridDim.x * blockDim.x) {
        const size_t i = (size_t)list[r];
        double* row = msg + kDomHeader + (size_t)r * kDomFullRow;
        row[0] = x[3 * i] + sx; row[1] = x[3 * i + 1] + sy; row[2] = x[3 * i + 2] + sz;
        row[3] = v[3 * i]; row[4] = v[3 * i + 1]; row[5] = v[3 * i + 2];
        row[6] = with_force ? f[3 * i] : 0.0; row[7] = with_force ? f[3 * i + 1] : 0.0; row[8] = with_force ? f[3 * i + 2] : 0.0;
        row[9] = (double)types[i];
        row[10] = (double)tag[i];
    }
}

// full rows of a message -> slots [base, base + count) of the state, base = dom[kDomNLocal] (bumped by k_dom_bump)
// The header comes from a peer: a count that is negative, not finite or above the capacity both sides agreed on
// (another build, a stale buffer) must not drive reads past the end of the message -- clamp and flag.
__device__ __forceinline__ int dom_msg_rows(const double* __restrict__ msg, int cap_rows, bool* bad) {
    const double h = msg[0];
    *bad = !(h >= 0.0 && h <= (double)cap_rows);
    return *bad ? (h > 0.0 ? cap_rows : 0) : (int)h;  // NaN fails both comparisons: bad, 0 rows
}

__global__ void k_dom_append(const double* __restrict__ msg, int cap_rows, const int* __restrict__ dom, int n_cap,
                             double* __restrict__ x, double* __restrict__ v, double* __restrict__ f,
                             int* __restrict__ types, long long* __restrict__ tag, int* __restrict__ flags) {
    const int base = dom[kDomNLocal];
    bool bad;
    int cnt = dom_msg_rows(msg, cap_rows, &bad);
    if (bad && blockIdx.x == 0 && threadIdx.x == 0) atomicOr(flags, kFlagDomainOverflow);
    if (base + cnt > n_cap) {
        cnt = max(0, n_cap - base);
        if (blockIdx.x == 0 && threadIdx.x == 0) atomicOr(flags, kFlagDomainOverflow);
    }
    for (int r = blockIdx.x * blockDim.x + threadIdx.x; r < cnt; r += gridDim.x * blockDim.x) {
        const double* row = msg + kDomHeader + (size_t)r * kDomFullRow;
        const size_t i = (size_t)(base + r);
#pragma unroll
        for (int d = 0; d < 3; d++) { x[3 * i + d] = row[d]; v[3 * i + d] = row[3 + d]; f[3 * i + d] = row[6 + d]; }
        types[i] = (int)row[9];
        tag[i] = (long long)row[10];
    }
}

// after k_dom_append: record where the rows went and move the end of the local set (and of the owned set for arrivals)
__global__ void k_dom_bump(const double* __restrict__ msg, int cap_rows, int* __restrict__ dom, int n_cap, int slot,
                           int owned) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    const int base = dom[kDomNLocal];
    bool bad;
    const int cnt = max(0, min(dom_msg_rows(msg, cap_rows, &bad), n_cap - base));
    if (slot >= 0) { dom[kDomRecvOff + slot] = base; dom[kDomRecvCnt + slot] = cnt; }
    dom[kDomNLocal] = base + cnt;
    if (owned) dom[kDomNOwned] = base + cnt;
}

// the atoms that stay, in order -> scratch copies; then back to the front of the state arrays
__global__ void k_dom_gather_stay(const int* __restrict__ list, const int* __restrict__ dom, const double* __restrict__ x,
                                  const double* __restrict__ v, const double* __restrict__ f,
                                  const int* __restrict__ types, const long long* __restrict__ tag,
                                  double* __restrict__ tmp /*[n][11]*/) {
    if (dom[kDomTot] + dom[kDomTot + 1] == 0) return;  // nobody leaves: the atoms that stay are already in place
    const int cnt = dom[kDomTot + 2];
    for (int r = blockIdx.x * blockDim.x + threadIdx.x; r < cnt; r += gridDim.x * blockDim.x) {
        const size_t i = (size_t)list[r];
        double* row = tmp + (size_t)r * kDomFullRow;
#pragma unroll
        for (int d = 0; d < 3; d++) { row[d] = x[3 * i + d]; row[3 + d] = v[3 * i + d]; row[6 + d] = f[3 * i + d]; }
        row[9] = (double)types[i];
        row[10] = (double)tag[i];
    }
}
__global__ void k_dom_scatter_stay(const int* __restrict__ dom, const double* __restrict__ tmp, double* __restrict__ x,
                                   double* __restrict__ v, double* __restrict__ f, int* __restrict__ types,
                                   long long* __restrict__ tag) {
    if (dom[kDomTot] + dom[kDomTot + 1] == 0) return;
    const int cnt = dom[kDomTot + 2];
    for (int r = blockIdx.x * blockDim.x + threadIdx.x; r < cnt; r += gridDim.x * blockDim.x) {
        const double* row = tmp + (size_t)r * kDomFullRow;
        const size_t i = (size_t)r;
#pragma unroll
        for (int d = 0; d < 3; d++) { x[3 * i + d] = row[d]; v[3 * i + d] = row[3 + d]; f[3 * i + d] = row[6 + d]; }
        types[i] = (int)row[9];
        tag[i] = (long long)row[10];
    }
}
__global__ void k_dom_set_counts(int* __restrict__ dom, int from_slot, int to_local, int to_owned) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    const int v = dom[from_slot];
    if (to_local) dom[kDomNLocal] = v;
    if (to_owned) dom[kDomNOwned] = v;
}

// ---- per MD step: fixed lists, counts known to the host
__global__ void k_dom_pack_fwd(const int* __restrict__ list, int cnt, double sx, double sy, double sz,
                               const double* __restrict__ x, const double* __restrict__ v, const double* __restrict__ f,
                               double* __restrict__ msg) {
    if (blockIdx.x == 0 && threadIdx.x == 0) msg[0] = (double)cnt;
    for (int r = blockIdx.x * blockDim.x + threadIdx.x; r < cnt; r += gridDim.x * blockDim.x) {
        const size_t i = (size_t)list[r];
        double* row = msg + kDomHeader + (size_t)r * kDomFwdRow;
        row[0] = x[3 * i] + sx; row[1] = x[3 * i + 1] + sy; row[2] = x[3 * i + 2] + sz;
#pragma unroll
        for (int d = 0; d < 3; d++) { row[3 + d] = v[3 * i + d]; row[6 + d] = f[3 * i + d]; }
    }
}
__global__ void k_dom_unpack_fwd(const double* __restrict__ msg, int off, int cnt, double* __restrict__ x,
                                 double* __restrict__ v, double* __restrict__ f, int* __restrict__ flags) {
    if (blockIdx.x == 0 && threadIdx.x == 0 && (int)msg[0] != cnt) atomicOr(flags, kFlagDomainOverflow);  // peer out of step
    for (int r = blockIdx.x * blockDim.x + threadIdx.x; r < cnt; r += gridDim.x * blockDim.x) {
        const double* row = msg + kDomHeader + (size_t)r * kDomFwdRow;
        const size_t i = (size_t)(off + r);
#pragma unroll
        for (int d = 0; d < 3; d++) { x[3 * i + d] = row[d]; v[3 * i + d] = row[3 + d]; f[3 * i + d] = row[6 + d]; }
    }
}

// ------------------------------------------------------------------ host-side drivers
static int dom_grid(int n) { return std::max(1, std::min((n + 255) / 256, 148 * 8)); }

void dom_select(Launcher& L, const Workspace& ws, const DomSel& s, int n_bound, int* list_lo, int* list_hi,
                int* list_stay, int cap) {  // the stay list (if any) holds up to n_bound entries
    const int nb = std::max(1, (n_bound + kDomBlock - 1) / kDomBlock);
    int* blk = ws.cell_cnt;  // scratch (free between evaluations): 3 nb ints
    L.launch(k_dom_count, dim3(nb), dim3(kDomBlock), 0, s, (const int*)ws.dom, (const double*)ws.x, blk);
    L.launch(k_dom_scan, dim3(1), dim3(1024), 0, nb, blk, ws.dom);
    L.launch(k_dom_write, dim3(nb), dim3(kDomBlock), 0, s, (const int*)ws.dom, (const double*)ws.x, (const int*)blk,
             list_lo, list_hi, list_stay, cap, n_bound, ws.flags);
}

void dom_commit_lists(Launcher& L, const Workspace& ws, int slot_lo, int slot_hi, int cap) {
    L.launch(k_dom_commit_lists, dim3(1), dim3(32), 0, ws.dom, slot_lo, slot_hi, cap);
}

void dom_pack_full(Launcher& L, const Workspace& ws, const int* list, int cnt_slot, const double shift[3],
                   bool with_force, double* msg, int cap_rows) {
    L.launch(k_dom_pack_full, dim3(dom_grid(cap_rows)), dim3(256), 0, list, (const int*)ws.dom, cnt_slot, shift[0],
             shift[1], shift[2], (const double*)ws.x, (const double*)ws.v, (const double*)ws.f, (const int*)ws.types,
             (const long long*)ws.tag, with_force ? 1 : 0, msg, cap_rows, ws.flags);
}

void dom_append(Launcher& L, const Workspace& ws, const double* msg, int n_cap, int max_rows, int slot, bool owned) {
    L.launch(k_dom_append, dim3(dom_grid(max_rows)), dim3(256), 0, msg, max_rows, (const int*)ws.dom, n_cap, ws.x, ws.v,
             ws.f, ws.types, ws.tag, ws.flags);
    L.launch(k_dom_bump, dim3(1), dim3(32), 0, msg, max_rows, ws.dom, n_cap, slot, owned ? 1 : 0);
}

void dom_compact_stay(Launcher& L, const Workspace& ws, const int* list_stay, int n_bound) {
    double* tmp = ws.pairf;  // scratch (free between evaluations): 11 doubles per atom of the 3 mmax it holds
    L.launch(k_dom_gather_stay, dim3(dom_grid(n_bound)), dim3(256), 0, list_stay, (const int*)ws.dom,
             (const double*)ws.x, (const double*)ws.v, (const double*)ws.f, (const int*)ws.types,
             (const long long*)ws.tag, tmp);
    L.launch(k_dom_scatter_stay, dim3(dom_grid(n_bound)), dim3(256), 0, (const int*)ws.dom, (const double*)tmp, ws.x,
             ws.v, ws.f, ws.types, ws.tag);
    L.launch(k_dom_set_counts, dim3(1), dim3(32), 0, ws.dom, kDomTot + 2, 1, 1);
}

void dom_set_counts(Launcher& L, const Workspace& ws, int from_slot, bool to_local, bool to_owned) {
    L.launch(k_dom_set_counts, dim3(1), dim3(32), 0, ws.dom, from_slot, to_local ? 1 : 0, to_owned ? 1 : 0);
}

void dom_pack_fwd(Launcher& L, const Workspace& ws, const int* list, int cnt, const double shift[3], double* msg) {
    L.launch(k_dom_pack_fwd, dim3(dom_grid(cnt)), dim3(256), 0, list, cnt, shift[0], shift[1], shift[2],
             (const double*)ws.x, (const double*)ws.v, (const double*)ws.f, msg);
}

void dom_unpack_fwd(Launcher& L, const Workspace& ws, const double* msg, int off, int cnt) {
    L.launch(k_dom_unpack_fwd, dim3(dom_grid(cnt)), dim3(256), 0, msg, off, cnt, ws.x, ws.v, ws.f, ws.flags);
}

}  // namespace flare
