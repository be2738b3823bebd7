// flare_api.cu -- the C ABI of include/flare_b200.h: context, workspace carving, the step scheduler
// that orders the kernels of steps a1-a9 on the caller's stream, and the host-buffer entry points.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

#include "../../include/flare_b200.h"
#include "kernels.cuh"

using namespace flare;

namespace {

constexpr double kKappa = 9.648533212331e-3;  // (eV/amu) in A^2/fs^2 (R13)

struct PhaseEvents {
    std::vector<cudaEvent_t> start, stop;
    size_t used = 0;
    int64_t launches = 0;
};

}  // namespace

struct flare_ctx {
    int device = 0;
    int sm_count = 148;
    Basis bs{};
    YNorm yn{};
    std::vector<double> mass;
    bool has_sigma = false;
    // model on device: two group sets are built at create time, [0] dense (one group per central species),
    // [1] species-sparse (one group per (central species, neighbour-species mask)); the active one
    // is mirrored into groups / d_groups / n_groups / max_ntn / ld
    std::vector<void*> dev_allocs;
    struct GroupSet {
        std::vector<GroupDesc> groups;        // host copy (device pointers inside)
        std::vector<std::vector<int>> comps;  // per group: dense component index of each compacted component
        GroupDev* d_groups = nullptr;
        int n_groups = 0, max_ntn = 0, ld = 0;
    } sets[2];
    bool have_sparse = false;
    std::vector<GroupDesc> groups;
    GroupDev* d_groups = nullptr;
    int n_groups = 0;
    int max_ntn = 0;
    int ld = 0;
    double* d_accel = nullptr;  // [S] 0.5 dt kappa / m
    double* d_mass = nullptr;   // [S] amu
    double skin = 0.4;          // Angstrom; 0 = rebuild the neighbour list at every evaluation
    bool list_valid = false;    // a skin list exists for the bound workspace and the current grid
    bool last_eval_var = false; // the last evaluation produced variances (v_s is meaningful)
    bool pairf_valid = false;   // an evaluation has been run since flare_bind (pair forces, neighbour list valid)
    double accel_dt = -1.0;
    std::vector<double> h_accel;
    // options
    int mmax = 48;
    int64_t chunk_opt = 0;
    int timing = 0;
    int sparse = 0;
    // binding
    int64_t n = -1;      // atoms the kernels work on
    int64_t n_cap = -1;  // atoms the workspace was carved for (n <= n_cap; they differ only in domain mode)
    // domain decomposition (flare_domain_*): host mirrors of the device counters after flare_domain_commit
    bool dom_active = false;
    double dom_trigger = 0.0;       // displacement since the last rebuild that raises the rebuild signal
    double dom_limit = 0.0;         // displacement since the last rebuild that is an error (0: not checked)
    double dom_shift[4][3]{};       // frame shift of the send lists x-lo, x-hi, y-lo, y-hi
    int dom_send[4]{}, dom_recv_cnt[4]{}, dom_recv_off[4]{};
    int64_t dom_n_owned = 0;
    int dom_list_cap = 0;
    Workspace ws{};
    cudaStream_t stream = nullptr;
    int chunk_cap = 0;
    int n_cells_cap = 0;
    Grid grid{};
    bool have_grid = false;
    bool state_set = false;
    bool forces_valid = false;
    bool var_valid = false;
    double box[9]{};
    int pbc[3]{};
    // bookkeeping
    int64_t launches = 0;
    LaunchCache launch_cache;  // per-context (= per-device) kernel attributes and occupancies
    // CUDA graph of one MD step (small systems: the step is launch-latency bound)
    int graph_opt = -1;                 // FLARE_OPT_GRAPH: -1 automatic, 0 never, 1 always
    cudaStream_t cap_stream = nullptr;  // capture happens on library-owned streams (the bound one may be the legacy
    cudaStream_t body_stream = nullptr; // default stream, which cannot be captured); replay goes to the bound stream
    cudaGraph_t step_graph = nullptr;
    cudaGraphExec_t step_exec = nullptr;
    struct StepKey {
        double dt = 0.0, T = 0.0, tau = 0.0;
        int var = 0;
        bool operator==(const StepKey& o) const { return dt == o.dt && T == o.T && tau == o.tau && var == o.var; }
    } graph_key, plain_key;
    bool plain_stepped = false;         // a plain (uncaptured) step with plain_key has run since the last invalidation
    bool graph_broken = false;          // capture failed once: stay on plain launches
    bool capturing = false;
    int64_t graph_launches = 0;         // kernels per replay
    int64_t graph_replays = 0;
    // side stream on which the per-group launches of the small groups run beside the large one (kernels.cuh)
    cudaStream_t side_stream = nullptr;
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
    int* h_group_start = nullptr;  // pinned [kMaxGroups + 1]: group offsets of the previous evaluation (scheduling hint)
    PhaseEvents phases[FLARE_N_PHASES];
    std::string err;
};

namespace {

Launcher make_launcher(flare_ctx* c) {
    Launcher L;
    L.stream = c->stream;
    L.launch_count = &c->launches;
    L.cache = &c->launch_cache;
    if (c->side_stream && c->h_group_start && c->n_groups > 1) {
        L.side = c->side_stream;
        L.ev_fork = c->ev_fork;
        L.ev_join = c->ev_join;
        int best = 0;
        for (int g = 0; g < c->n_groups; g++) {
            const int rows = c->h_group_start[g + 1] - c->h_group_start[g];
            if (rows > best) { best = rows; L.big_group = g; }
        }
    }
    return L;
}

// the captured step bakes in pointers, the grid, options and dt: anything that changes them drops it
void drop_step_graph(flare_ctx* c) {
    if (c->step_exec) cudaGraphExecDestroy(c->step_exec);
    if (c->step_graph) cudaGraphDestroy(c->step_graph);
    c->step_exec = nullptr;
    c->step_graph = nullptr;
    c->plain_stepped = false;
}

int fail(flare_ctx* c, int code, const std::string& msg) {
    if (c) c->err = msg;
    return code;
}

int cuda_fail(flare_ctx* c, cudaError_t e, const char* where) {
    return fail(c, FLARE_ERR_CUDA, std::string(where) + ": " + cudaGetErrorString(e));
}

#define FLARE_CUDA(ctx, call)                                         \
    do {                                                              \
        cudaError_t e__ = (call);                                     \
        if (e__ != cudaSuccess) return cuda_fail(ctx, e__, #call);    \
    } while (0)

struct PhaseScope {
    flare_ctx* c;
    int phase;
    int64_t l0;
    PhaseScope(flare_ctx* ctx, int p) : c(ctx), phase(p), l0(ctx->launches) {
        if (!c->timing || c->capturing) return;
        PhaseEvents& pe = c->phases[phase];
        if (pe.used == pe.start.size()) {
            cudaEvent_t a, b;
            cudaEventCreate(&a);
            cudaEventCreate(&b);
            pe.start.push_back(a);
            pe.stop.push_back(b);
        }
        cudaEventRecord(pe.start[pe.used], c->stream);
    }
    ~PhaseScope() {
        if (!c->timing || c->capturing) return;
        PhaseEvents& pe = c->phases[phase];
        cudaEventRecord(pe.stop[pe.used], c->stream);
        pe.used++;
        pe.launches += c->launches - l0;
    }
};

int round_up(int v, int m) { return (v + m - 1) / m * m; }

// the skin list needs one 64-bit hit mask per atom: rows longer than 64 switch it off
double eff_skin(const flare_ctx* c) { return c->mmax <= kSkinStride ? c->skin : 0.0; }

// choose the tile width (in n8 blocks): the WIDEST one that pads the matrix by at most 5 % (wide tiles reuse the
// B rows more and leave fewer partial row-dots: K = 544 -> 5 tiles of 112, not 17 of 32); if none, the least padding
void choose_tiles(int K, int& nb, int& ntn) {
    // even widths only: a tile then starts on a 16-column super-block (the variance tiles' triangular schedule)
    static const int cand[] = {18, 16, 14, 12, 10, 8, 6, 4, 2};
    const int n8 = K / 8;
    long best = -1;
    nb = 2; ntn = (n8 + 1) / 2;
    for (int c : cand) {
        const int t = (n8 + c - 1) / c;
        const long width = (long)t * c;
        if (width * 100 <= (long)n8 * 105) { nb = c; ntn = t; return; }
        if (best < 0 || width < best) { best = width; nb = c; ntn = t; }
    }
}

template <class T>
int upload(flare_ctx* c, const std::vector<T>& h, T** d_out) {
    void* d = nullptr;
    FLARE_CUDA(c, cudaMalloc(&d, std::max<size_t>(sizeof(T) * h.size(), 16)));
    c->dev_allocs.push_back(d);
    if (!h.empty()) FLARE_CUDA(c, cudaMemcpy(d, h.data(), sizeof(T) * h.size(), cudaMemcpyHostToDevice));
    *d_out = reinterpret_cast<T*>(d);
    return FLARE_OK;
}

// padded, symmetrised copy of the sub-matrix of `m` (P x P, row-major) on the components `comp`
std::vector<double> pack_matrix(const double* m, int P, const std::vector<int>& comp, int K, int rows) {
    std::vector<double> out((size_t)rows * K, 0.0);
    const int n = (int)comp.size();
    for (int a = 0; a < n; a++)
        for (int b = 0; b < n; b++)
            out[(size_t)a * K + b] = 0.5 * (m[(size_t)comp[a] * P + comp[b]] + m[(size_t)comp[b] * P + comp[a]]);
    return out;
}

void activate_groups(flare_ctx* c, int sparse) {
    const flare_ctx::GroupSet& gs = c->sets[sparse];
    c->sparse = sparse;
    c->groups = gs.groups;
    c->d_groups = gs.d_groups;
    c->n_groups = gs.n_groups;
    c->max_ntn = gs.max_ntn;
    c->ld = gs.ld;
    c->bs.Pld = gs.ld;
}

int build_groups(flare_ctx* c, const double* beta, const double* sigma, int sparse) {
    const Basis& bs = c->bs;
    const int S = bs.S, L = bs.l_max + 1, Nv = bs.Nv, P = bs.P;
    flare_ctx::GroupSet& set = c->sets[sparse];
    set.n_groups = sparse ? S * (1 << S) : S;
    set.groups.assign(set.n_groups, GroupDesc{});
    set.comps.assign(set.n_groups, {});
    std::vector<GroupDev> gdev(set.n_groups);
    set.max_ntn = 0;
    set.ld = 16;
    for (int gi = 0; gi < set.n_groups; gi++) {
        const int s = sparse ? gi / (1 << S) : gi;
        const unsigned mask = sparse ? (unsigned)(gi % (1 << S)) : ((1u << S) - 1u);
        // (nu1 <= nu2) pairs whose radial channels both belong to species present in the mask;
        // component p = q*L + l keeps the dense order (nu1, nu2, l) of R4 restricted to those pairs
        std::vector<int> comp, table, lut((size_t)Nv * Nv, -1);
        for (int v1 = 0, dense_q = 0; v1 < Nv; v1++)
            for (int v2 = v1; v2 < Nv; v2++, dense_q++) {
                const int s1 = v1 / bs.n_max, s2 = v2 / bs.n_max;
                if (!(((mask >> s1) & 1u) && ((mask >> s2) & 1u))) continue;
                lut[(size_t)v1 * Nv + v2] = lut[(size_t)v2 * Nv + v1] = (int)table.size();
                table.push_back(v1 | (v2 << 8));
                for (int l = 0; l < L; l++) comp.push_back(dense_q * L + l);
            }
        GroupDesc& gd = set.groups[gi];
        gd.P = (int)comp.size();
        gd.mask = mask;
        gd.sidx = 0;
        for (int sp = 0, rank = 0; sp < kMaxSpecies; sp++) {
            const bool in = sp < S && ((mask >> sp) & 1u);
            gd.sidx |= (unsigned)(in ? rank : 15) << (4 * sp);
            if (in) rank++;
            gd.nsp = rank;
        }
        gd.Nc = gd.nsp * bs.n_max;
        set.comps[gi] = comp;
        if (gd.P == 0) { gdev[gi] = GroupDev{0, 0, 0, 0, nullptr, nullptr}; continue; }
        gd.K = round_up(gd.P, 16);
        choose_tiles(gd.K, gd.nb, gd.ntn);
        const int rows = gd.ntn * gd.nb * 8;
        double* d = nullptr;
        int rc = upload(c, pack_matrix(beta + (size_t)s * P * P, P, comp, gd.K, rows), &d);
        if (rc) return rc;
        gd.beta = d;
        if (sigma) {
            rc = upload(c, pack_matrix(sigma + (size_t)s * P * P, P, comp, gd.K, rows), &d);
            if (rc) return rc;
            gd.sigma = d;
        }
        int* dt = nullptr;
        rc = upload(c, table, &dt);
        if (rc) return rc;
        gd.table = dt;
        rc = upload(c, lut, &dt);
        if (rc) return rc;
        gd.lut = dt;
        gdev[gi] = GroupDev{gd.P, gd.K, gd.ntn, 0, gd.table, gd.lut};
        set.max_ntn = std::max(set.max_ntn, gd.ntn);
        set.ld = std::max(set.ld, gd.K);
    }
    return upload(c, gdev, &set.d_groups);
}

// ---------------------------------------------------------------- workspace layout
struct Carver {
    char* base;
    size_t off = 0;
    template <class T>
    T* take(size_t count) {
        off = (off + 255) & ~(size_t)255;
        T* p = base ? reinterpret_cast<T*>(base + off) : nullptr;
        off += sizeof(T) * count;
        return p;
    }
};

// Small systems: the tile kernel of the large matrices (K > 144) is latency-bound there -- a 64 x 112 tile is
// 34 slabs of K = 544 run back to back on one SM -- so below kNarrowAtoms atoms the tiles are 16 columns wide (nb = 2,
// K / 16 tiles per matrix): many short tiles on many SMs.  The matrices keep their layout (rows = columns of the symmetric
// matrix, K of them are always there); only the number of partial row-dots per row grows, which small systems can afford.
constexpr int64_t kNarrowAtoms = 8192;
constexpr int kResidentK = 144;  // largest K of the resident-matrix kernel (qform.cu)

int eff_max_ntn(const flare_ctx* c, bool narrow) {
    int m = 0;
    for (const GroupDesc& g : c->sets[c->sparse].groups) m = std::max(m, (narrow && g.K > kResidentK) ? g.K / 16 : g.ntn);
    return m;
}

void apply_tiling(flare_ctx* c, bool narrow) {
    const flare_ctx::GroupSet& gs = c->sets[c->sparse];
    for (int g = 0; g < gs.n_groups; g++) {
        c->groups[g].nb = gs.groups[g].nb;
        c->groups[g].ntn = gs.groups[g].ntn;
        if (narrow && gs.groups[g].K > kResidentK) { c->groups[g].nb = 2; c->groups[g].ntn = gs.groups[g].K / 16; }
    }
    c->max_ntn = eff_max_ntn(c, narrow);
}

int auto_chunk(const flare_ctx* c, int64_t n) {
    if (c->chunk_opt > 0) return (int)std::min<int64_t>(std::max<int64_t>(c->chunk_opt, 1), std::max<int64_t>(n, 1));
    const double per_row = 8.0 * (c->bs.NvL2 + 2.0 * c->ld + 1 + 2.0 * c->max_ntn);
    int64_t rows = (int64_t)(16.0 * 1024 * 1024 * 1024 / per_row);  // 16 GiB of chunk intermediates (of 180 GB)
    rows = std::max<int64_t>(rows, 16384);
    return (int)std::max<int64_t>(1, std::min<int64_t>(rows, n));
}

size_t carve(const flare_ctx* c, int64_t n, char* base, Workspace* ws, int* chunk_out, int* cells_out) {
    Carver cv{base};
    const size_t N = (size_t)std::max<int64_t>(n, 1);
    const int chunk = auto_chunk(c, n);
    const size_t cells = std::max<size_t>(4096, 2 * N);
    Workspace w;
    w.x = cv.take<double>(3 * N);
    w.v = cv.take<double>(3 * N);
    w.f = cv.take<double>(3 * N);
    w.e = cv.take<double>(N);
    w.var = cv.take<double>(N);
    w.types = cv.take<int>(N);
    w.flags = cv.take<int>(4);
    w.cell_cnt = cv.take<int>(cells);
    w.cell_start = cv.take<int>(cells + 1);
    w.scan_tmp = cv.take<int>(cells / 1024 + 2);
    w.cell_of = cv.take<int>(N);
    w.rank_in_cell = cv.take<int>(N);
    w.order = cv.take<int>(N);
    w.atoms = cv.take<AtomS>(N);
    w.nbr_cnt = cv.take<int>(N);
    w.nbr_idx = cv.take<int>(N * c->mmax);
    w.rev = cv.take<unsigned char>(N * c->mmax);
    w.nmask = cv.take<unsigned char>(N);
    w.group_hist = cv.take<int>((N / 1024 + 1) * (size_t)c->n_groups);
    w.group_start = cv.take<int>(c->n_groups + 1);
    w.row_of = cv.take<int>(N);
    w.gid = cv.take<unsigned char>(N);
    w.atom_of_row = cv.take<int>(N);
    if (eff_skin(c) > 0.0) {
        w.skin_cnt = cv.take<int>(N);
        w.skin_idx = cv.take<int>(N * kSkinStride);
        w.skin_rev = cv.take<unsigned char>(N * kSkinStride);
        w.ref = cv.take<AtomS>(N);
        w.hitmask = cv.take<unsigned long long>(N);
        w.skin_gate = cv.take<int>(4 + kMaxSpecies);  // gate, rebuild count, -, -, per-species max displacement
    }
    w.pairf = cv.take<double>(N * c->mmax * 3);
    w.e_s = cv.take<double>(N);
    w.v_s = cv.take<double>(N);
    w.A = cv.take<double>((size_t)chunk * c->bs.NvL2);
    w.Bh = cv.take<double>((size_t)chunk * c->ld);
    w.W = cv.take<double>((size_t)chunk * c->ld);
    w.nrm = cv.take<double>(chunk);
    w.part = cv.take<double>((size_t)2 * std::max(eff_max_ntn(c, n <= kNarrowAtoms), 1) * chunk);
    w.red = cv.take<double>((size_t)kRedBlocksMax * 9);
    w.scal = cv.take<double>(16);
    w.ascal = cv.take<unsigned long long>(18);
    w.qf_counter = cv.take<int>(3 * kMaxGroups);
    w.tag = cv.take<long long>(N);
    w.dom = cv.take<int>(kDomInts);
    w.send_idx = cv.take<int>(4 * (N / 2 + 1024));
    w.dom_ref = cv.take<double>(3 * N);
    if (ws) *ws = w;
    if (chunk_out) *chunk_out = chunk;
    if (cells_out) *cells_out = (int)std::min<size_t>(cells, 0x7fffffff);
    return ((cv.off + 255) & ~(size_t)255) + 256;
}

// ---------------------------------------------------------------- box -> cell grid (R7)
int setup_grid(flare_ctx* c, const double box[9], const int pbc[3]) {
    if (!box || !pbc) return fail(c, FLARE_ERR_INVALID_ARG, "box/pbc is null");
    if (c->have_grid && memcmp(c->box, box, sizeof(double) * 9) == 0 && c->pbc[0] == (pbc[0] ? 1 : 0) &&
        c->pbc[1] == (pbc[1] ? 1 : 0) && c->pbc[2] == (pbc[2] ? 1 : 0))
        return FLARE_OK;  // same cell as before: the grid (and whatever was built on it) stands
    for (int i = 0; i < 9; i++)
        if (!std::isfinite(box[i])) return fail(c, FLARE_ERR_INVALID_ARG, "box has a non-finite entry");
    if (box[1] != 0 || box[2] != 0 || box[3] != 0 || box[5] != 0 || box[6] != 0 || box[7] != 0)
        return fail(c, FLARE_ERR_UNSUPPORTED_BOX, "only orthorhombic cells are supported (R7)");
    if (!(box[0] > 0 && box[4] > 0 && box[8] > 0)) return fail(c, FLARE_ERR_INVALID_ARG, "box lengths must be > 0");
    double rcmax = 0;
    for (int i = 0; i < c->bs.S * c->bs.S; i++) rcmax = std::max(rcmax, c->bs.rc[i]);
    Grid g{};
    for (int d = 0; d < 3; d++) {
        g.L[d] = box[4 * d];
        g.half[d] = 0.5 * g.L[d];
        g.pbc[d] = pbc[d] ? 1 : 0;
        if (g.pbc[d] && g.L[d] < 2.0 * rcmax)
            return fail(c, FLARE_ERR_BOX_TOO_SMALL, "a periodic box length is < 2 max r_cut (R7)");
        int nc = (int)std::floor(g.L[d] / ((rcmax + eff_skin(c)) * (1.0 + 1e-9)));  // cells hold the skin list's cutoff
        g.nc[d] = std::max(1, nc);
    }
    // keep the number of cells within what the workspace was sized for
    while ((double)g.nc[0] * g.nc[1] * g.nc[2] > (double)c->n_cells_cap) {
        int dmax = 0;
        for (int d = 1; d < 3; d++) if (g.nc[d] > g.nc[dmax]) dmax = d;
        g.nc[dmax] = std::max(1, (int)(g.nc[dmax] * 0.8));
    }
    for (int d = 0; d < 3; d++) g.inv_cw[d] = (double)g.nc[d] / g.L[d];
    // dimension with the fewest cells runs fastest (a thin slab's z column becomes contiguous)
    int ord[3] = {0, 1, 2};
    std::sort(ord, ord + 3, [&](int a, int b) { return g.nc[a] < g.nc[b] || (g.nc[a] == g.nc[b] && a > b); });
    g.fast = ord[0]; g.slow0 = ord[1]; g.slow1 = ord[2];
    g.stride[g.fast] = 1;
    g.stride[g.slow0] = g.nc[g.fast];
    g.stride[g.slow1] = g.nc[g.fast] * g.nc[g.slow0];
    g.n_cells = g.nc[0] * g.nc[1] * g.nc[2];
    if (!c->have_grid || memcmp(&c->grid, &g, sizeof(Grid)) != 0) { c->list_valid = false; drop_step_graph(c); }  // new box: new list
    c->grid = g;
    c->have_grid = true;
    memcpy(c->box, box, sizeof(double) * 9);
    for (int d = 0; d < 3; d++) c->pbc[d] = g.pbc[d];
    return FLARE_OK;
}

// ---------------------------------------------------------------- one evaluation (steps a1-a8)
int evaluate(flare_ctx* c, Launcher& L, const double* pos, const int* types, double* e_out, double* f_out,
             double* var_out) {
    const int n = (int)c->n;
    const bool want_var = (var_out != nullptr) && c->has_sigma;
    if (var_out && !c->has_sigma) return fail(c, FLARE_ERR_INVALID_ARG, "variance requested but the model has no sigma");
    if (n == 0) return FLARE_OK;
    {
        PhaseScope ps(c, FLARE_PHASE_NEIGHBOR);
        build_neighbors(L, c->grid, c->bs, c->ws, n, pos, types, c->mmax, c->sparse, c->n_groups, eff_skin(c),
                        c->list_valid, c->dom_active ? c->dom_trigger : 0.0,
                        c->dom_active ? c->dom_limit : 0.0);
        if (eff_skin(c) > 0.0) c->list_valid = true;
        // group sizes of this evaluation -> pinned host memory, read (without waiting) when the NEXT evaluation is enqueued
        if (c->h_group_start && !c->capturing && L.err == cudaSuccess)
            cudaMemcpyAsync(c->h_group_start, c->ws.group_start, sizeof(int) * (c->n_groups + 1), cudaMemcpyDeviceToHost, L.stream);
    }
    for (int row0 = 0; row0 < n; row0 += c->chunk_cap) {
        const int nrows = std::min(c->chunk_cap, n - row0);
        {
            PhaseScope ps(c, FLARE_PHASE_DESCRIPTOR);
            run_descriptors(L, c->grid, c->bs, c->yn, c->ws, c->mmax, c->groups.data(), c->n_groups, row0, nrows,
                            c->ws.Bh, c->ld, c->ws.nrm, true);
        }
        {
            PhaseScope ps(c, FLARE_PHASE_QFORM);
            run_qform(L, c->ws, c->groups.data(), c->n_groups, row0, nrows, c->ld, c->chunk_cap, want_var, c->sm_count);
        }
        {
            PhaseScope ps(c, FLARE_PHASE_BACKPROP);
            run_backprop(L, c->grid, c->bs, c->yn, c->ws, c->mmax, c->groups.data(), c->n_groups, row0, nrows, c->ld,
                         c->chunk_cap, c->max_ntn, want_var);
        }
    }
    {
        PhaseScope ps(c, FLARE_PHASE_GATHER);
        run_gather(L, c->ws, n, c->mmax, e_out, f_out, var_out);
    }
    if (L.err != cudaSuccess) return cuda_fail(c, L.err, L.err_where ? L.err_where : "launch");
    c->last_eval_var = want_var;
    c->pairf_valid = true;
    return FLARE_OK;
}

int need_bound(flare_ctx* c) {
    if (!c) return FLARE_ERR_INVALID_ARG;
    if (c->n < 0) return fail(c, FLARE_ERR_NOT_BOUND, "flare_bind has not been called");
    return FLARE_OK;
}

// Calls that take whole-system arrays sized by flare_bind's n_atoms.  In domain mode the context works on the local
// atoms (owned + ghosts, fewer than the bound capacity, in the rank's open frame) and tracks displacements against
// the last domain rebuild: a plain call would silently evaluate a truncated system with the caller's arrays read at
// the wrong length.  Refuse it; flare_bind ends domain mode.
int need_plain(flare_ctx* c, const char* what) {
    int rc = need_bound(c);
    if (rc) return rc;
    if (c->dom_active)
        return fail(c, FLARE_ERR_INVALID_ARG, std::string(what) + ": the context is in domain mode (flare_domain_begin); "
                    "call flare_bind again to return to plain whole-system calls");
    return FLARE_OK;
}

}  // namespace

// ================================================================= C ABI
extern "C" {
#pragma GCC visibility push(default)

int flare_create(flare_ctx** out, int n_species, const double* mass_amu, int n_max, int l_max, const double* r_cut,
                 const double* beta, const double* sigma, int cuda_device) {
    if (!out) return FLARE_ERR_INVALID_ARG;
    *out = nullptr;
    if (!mass_amu || !r_cut || !beta) return FLARE_ERR_INVALID_ARG;
    if (n_species < 1 || n_species > kMaxSpecies) return FLARE_ERR_INVALID_ARG;
    if (n_max < 1 || n_max > kMaxNmax || l_max < 0 || l_max > kMaxLmax) return FLARE_ERR_UNSUPPORTED;
    if (n_species * n_max > 255) return FLARE_ERR_UNSUPPORTED;
    for (int a = 0; a < n_species; a++) {
        if (!(mass_amu[a] > 0)) return FLARE_ERR_INVALID_ARG;
        for (int b = 0; b < n_species; b++) {
            const double r = r_cut[a * n_species + b];
            if (!(r > 0) || !std::isfinite(r) || r != r_cut[b * n_species + a]) return FLARE_ERR_INVALID_ARG;  // R5
        }
    }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0 || cuda_device < 0 || cuda_device >= ndev)
        return FLARE_ERR_CUDA;  // no CPU fallback
    if (cudaSetDevice(cuda_device) != cudaSuccess) return FLARE_ERR_CUDA;
    flare_ctx* c = new (std::nothrow) flare_ctx();
    if (!c) return FLARE_ERR_CUDA;
    c->device = cuda_device;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, cuda_device) == cudaSuccess) c->sm_count = prop.multiProcessorCount;
    Basis& bs = c->bs;
    bs.S = n_species; bs.n_max = n_max; bs.l_max = l_max;
    bs.L2 = (l_max + 1) * (l_max + 1);
    bs.Nv = n_species * n_max;
    bs.NvL2 = bs.Nv * bs.L2;
    bs.P = bs.Nv * (bs.Nv + 1) / 2 * (l_max + 1);
    for (int i = 0; i < n_species * n_species; i++) { bs.rc[i] = r_cut[i]; bs.rc2[i] = r_cut[i] * r_cut[i]; bs.irc[i] = 1.0 / r_cut[i]; }
    c->mass.assign(mass_amu, mass_amu + n_species);
    c->has_sigma = sigma != nullptr;
    // K_lm sqrt(2 - delta_m0)
    for (int l = 0; l <= kMaxLmax; l++)
        for (int m = 0; m <= l; m++) {
            double ratio = 1.0;  // (l-m)!/(l+m)!
            for (int q = l - m + 1; q <= l + m; q++) ratio /= (double)q;
            double k = std::sqrt((2.0 * l + 1.0) / (4.0 * kPi) * ratio);
            if (m > 0) k *= std::sqrt(2.0);
            c->yn.k[l * (l + 1) / 2 + m] = k;
        }
    int rc = build_groups(c, beta, sigma, 0);
    c->have_sparse = n_species * (1 << n_species) <= kMaxGroups;
    if (rc == FLARE_OK && c->have_sparse) rc = build_groups(c, beta, sigma, 1);
    if (rc == FLARE_OK) activate_groups(c, c->have_sparse ? 1 : 0);  // species-sparse evaluation is the default
    if (rc == FLARE_OK) {
        void* d = nullptr;
        if (cudaMalloc(&d, sizeof(double) * kMaxSpecies) != cudaSuccess) rc = FLARE_ERR_CUDA;
        else { c->dev_allocs.push_back(d); c->d_accel = (double*)d; }
    }
    if (rc == FLARE_OK) {
        std::vector<double> hm(kMaxSpecies, 1.0);
        for (int s = 0; s < n_species; s++) hm[s] = mass_amu[s];
        rc = upload(c, hm, &c->d_mass);
    }
    if (rc == FLARE_OK) {
        if (cudaStreamCreateWithFlags(&c->side_stream, cudaStreamNonBlocking) != cudaSuccess ||
            cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&c->ev_join, cudaEventDisableTiming) != cudaSuccess ||
            cudaMallocHost(&c->h_group_start, sizeof(int) * (kMaxGroups + 1)) != cudaSuccess)
            rc = FLARE_ERR_CUDA;
        else
            memset(c->h_group_start, 0, sizeof(int) * (kMaxGroups + 1));
    }
    if (rc != FLARE_OK) { flare_destroy(c); return rc; }
    c->h_accel.assign(kMaxSpecies, 0.0);
    *out = c;
    return FLARE_OK;
}

void flare_destroy(flare_ctx* c) {
    if (!c) return;
    cudaSetDevice(c->device);
    drop_step_graph(c);
    if (c->side_stream) cudaStreamDestroy(c->side_stream);
    if (c->ev_fork) cudaEventDestroy(c->ev_fork);
    if (c->ev_join) cudaEventDestroy(c->ev_join);
    if (c->h_group_start) cudaFreeHost(c->h_group_start);
    if (c->cap_stream) cudaStreamDestroy(c->cap_stream);
    if (c->body_stream) cudaStreamDestroy(c->body_stream);
    for (void* p : c->dev_allocs) cudaFree(p);
    for (auto& pe : c->phases) {
        for (auto e : pe.start) cudaEventDestroy(e);
        for (auto e : pe.stop) cudaEventDestroy(e);
    }
    delete c;
}

int flare_num_descriptors(const flare_ctx* c) { return c ? c->bs.P : FLARE_ERR_INVALID_ARG; }

int flare_set_option(flare_ctx* c, int option, int64_t value) {
    if (!c) return FLARE_ERR_INVALID_ARG;
    switch (option) {
        case FLARE_OPT_MAX_NEIGHBORS:
            if (value < 1 || value > 255) return fail(c, FLARE_ERR_INVALID_ARG, "max neighbours must be in 1..255");
            c->mmax = (int)value; c->n = -1;
            return FLARE_OK;
        case FLARE_OPT_CHUNK_ATOMS:
            if (value < 0) return fail(c, FLARE_ERR_INVALID_ARG, "chunk must be >= 0");
            c->chunk_opt = value; c->n = -1;
            return FLARE_OK;
        case FLARE_OPT_TIMING:
            c->timing = value ? 1 : 0;
            return FLARE_OK;
        case FLARE_OPT_SKIN_MILLI_ANGSTROM:
            if (value < 0 || value > 4000) return fail(c, FLARE_ERR_INVALID_ARG, "skin must be in 0..4000 (1e-3 Angstrom)");
            c->skin = 1e-3 * (double)value; c->n = -1;
            return FLARE_OK;
        case FLARE_OPT_GRAPH:
            if (value < -1 || value > 1) return fail(c, FLARE_ERR_INVALID_ARG, "graph option must be -1, 0 or 1");
            c->graph_opt = (int)value;
            c->graph_broken = false;
            drop_step_graph(c);
            return FLARE_OK;
        case FLARE_OPT_SPECIES_SPARSE:
            if (value && !c->have_sparse)
                return fail(c, FLARE_ERR_UNSUPPORTED, "species-sparse mode needs S * 2^S <= 64 groups");
            activate_groups(c, value ? 1 : 0);
            c->n = -1;
            return FLARE_OK;
        default:
            return fail(c, FLARE_ERR_INVALID_ARG, "unknown option");
    }
}

int flare_get_option(const flare_ctx* c, int option, int64_t* value) {
    if (!c || !value) return FLARE_ERR_INVALID_ARG;
    switch (option) {
        case FLARE_OPT_MAX_NEIGHBORS: *value = c->mmax; return FLARE_OK;
        case FLARE_OPT_CHUNK_ATOMS: *value = c->n >= 0 ? c->chunk_cap : c->chunk_opt; return FLARE_OK;
        case FLARE_OPT_TIMING: *value = c->timing; return FLARE_OK;
        case FLARE_OPT_SPECIES_SPARSE: *value = c->sparse; return FLARE_OK;
        case FLARE_OPT_SKIN_MILLI_ANGSTROM: *value = (int64_t)std::llround(c->skin * 1e3); return FLARE_OK;
        case FLARE_OPT_GRAPH: *value = c->graph_opt; return FLARE_OK;
        case FLARE_OPT_GRAPH_REPLAYS: *value = c->graph_replays; return FLARE_OK;
        case FLARE_OPT_SKIN_REBUILDS: {
            *value = 0;
            if (c->n >= 0 && c->ws.skin_gate) {
                int h = 0;
                if (cudaStreamSynchronize(c->stream) != cudaSuccess ||
                    cudaMemcpy(&h, c->ws.skin_gate + 1, sizeof(int), cudaMemcpyDeviceToHost) != cudaSuccess)
                    return FLARE_ERR_CUDA;
                *value = h;
            }
            return FLARE_OK;
        }
        default: return FLARE_ERR_INVALID_ARG;
    }
}

size_t flare_workspace_bytes(const flare_ctx* c, int64_t n_atoms) {
    if (!c || n_atoms < 0 || n_atoms > 0x7fffffff / 4) return 0;
    return carve(c, n_atoms, nullptr, nullptr, nullptr, nullptr);
}

int flare_bind(flare_ctx* c, int64_t n_atoms, void* workspace, size_t bytes, void* cuda_stream) {
    if (!c) return FLARE_ERR_INVALID_ARG;
    if (n_atoms < 0 || n_atoms > 0x7fffffff / 4) return fail(c, FLARE_ERR_INVALID_ARG, "n_atoms out of range");
    if (!workspace) return fail(c, FLARE_ERR_INVALID_ARG, "workspace is null");
    if ((reinterpret_cast<uintptr_t>(workspace) & 255) != 0)
        return fail(c, FLARE_ERR_INVALID_ARG, "workspace must be 256-byte aligned");
    const size_t need = carve(c, n_atoms, nullptr, nullptr, nullptr, nullptr);
    if (bytes < need) return fail(c, FLARE_ERR_WORKSPACE_TOO_SMALL, "workspace smaller than flare_workspace_bytes");
    FLARE_CUDA(c, cudaSetDevice(c->device));
    carve(c, n_atoms, static_cast<char*>(workspace), &c->ws, &c->chunk_cap, &c->n_cells_cap);
    apply_tiling(c, n_atoms <= kNarrowAtoms);
    c->stream = static_cast<cudaStream_t>(cuda_stream);
    c->n = c->n_cap = n_atoms;
    c->dom_active = false;
    c->dom_limit = 0.0;
    c->dom_list_cap = (int)(std::max<int64_t>(n_atoms, 1) / 2 + 1024);
    c->state_set = c->forces_valid = c->var_valid = false;
    c->have_grid = false;
    c->pairf_valid = false;
    c->list_valid = false;
    drop_step_graph(c);
    FLARE_CUDA(c, cudaMemsetAsync(c->ws.flags, 0, sizeof(int) * 4, c->stream));
    FLARE_CUDA(c, cudaMemsetAsync(c->ws.scal, 0, sizeof(double) * 16, c->stream));  // thermostat xi = eta = 0
    if (c->ws.skin_gate) FLARE_CUDA(c, cudaMemsetAsync(c->ws.skin_gate, 0, sizeof(int) * 4, c->stream));
    FLARE_CUDA(c, cudaMemsetAsync(c->ws.dom, 0, sizeof(int) * kDomInts, c->stream));
    return FLARE_OK;
}

int flare_compute(flare_ctx* c, const double* pos, const int32_t* types, const double box[9], const int pbc[3],
                  double* e_out, double* f_out, double* var_out) {
    int rc = need_plain(c, "flare_compute");
    if (rc) return rc;
    if (c->n > 0 && (!pos || !types)) return fail(c, FLARE_ERR_INVALID_ARG, "pos/types is null");
    FLARE_CUDA(c, cudaSetDevice(c->device));
    rc = setup_grid(c, box, pbc);
    if (rc) return rc;
    Launcher L = make_launcher(c);
    return evaluate(c, L, pos, types, e_out, f_out, var_out);
}

int flare_check(flare_ctx* c) {
    int rc = need_bound(c);
    if (rc) return rc;
    FLARE_CUDA(c, cudaStreamSynchronize(c->stream));
    int flags[4] = {0, 0, 0, 0};
    FLARE_CUDA(c, cudaMemcpy(flags, c->ws.flags, sizeof(flags), cudaMemcpyDeviceToHost));
    if (flags[0]) {
        FLARE_CUDA(c, cudaMemset(c->ws.flags, 0, sizeof(flags)));
        // whatever went wrong, the kept candidate list and pair forces may be truncated or built from bad input:
        // the next evaluation rebuilds from scratch (and raises the error again if its cause persists)
        c->list_valid = false;
        c->pairf_valid = false;
        c->forces_valid = c->var_valid = false;
    }
    if (flags[0] & kFlagDomainOverflow)
        return fail(c, FLARE_ERR_WORKSPACE_TOO_SMALL, "domain decomposition: a message buffer, a send list or the bound capacity is too small (or a peer sent a message of another step)");
    if (flags[0] & kFlagHaloExceeded)
        return fail(c, FLARE_ERR_HALO_EXCEEDED, "domain decomposition: an atom has moved further since the last rebuild than flare_domain_set_limit allows; the ghost shell may have missed neighbours of owned atoms since then (widen the halo skin, lower the signal lag or the time step)");
    if (flags[0] & kFlagBadType) return fail(c, FLARE_ERR_INVALID_ARG, "a species index is outside 0..S-1");
    if (flags[0] & kFlagNonFinite) return fail(c, FLARE_ERR_NONFINITE, "non-finite position");
    if (flags[0] & kFlagNeighborOverflow)
        return fail(c, FLARE_ERR_NEIGHBOR_OVERFLOW, "an atom has more neighbours than FLARE_OPT_MAX_NEIGHBORS (or more than 64 candidates within r_cut + skin: lower FLARE_OPT_SKIN_MILLI_ANGSTROM)");
    if (flags[0] & kFlagNonFiniteResult)
        return fail(c, FLARE_ERR_NONFINITE, "a non-finite energy, force or variance was produced (atoms too close, or a blown-up step)");
    return FLARE_OK;
}

int flare_compute_host(flare_ctx* c, const double* pos, const int32_t* types, const double box[9], const int pbc[3],
                       double* e_out, double* f_out, double* var_out) {
    int rc = need_plain(c, "flare_compute_host");
    if (rc) return rc;
    const size_t n = (size_t)c->n;
    if (n > 0 && (!pos || !types)) return fail(c, FLARE_ERR_INVALID_ARG, "pos/types is null");
    FLARE_CUDA(c, cudaSetDevice(c->device));
    c->state_set = c->forces_valid = false;  // the state arrays serve as staging
    if (n > 0) {
        FLARE_CUDA(c, cudaMemcpyAsync(c->ws.x, pos, sizeof(double) * 3 * n, cudaMemcpyHostToDevice, c->stream));
        FLARE_CUDA(c, cudaMemcpyAsync(c->ws.types, types, sizeof(int) * n, cudaMemcpyHostToDevice, c->stream));
    }
    rc = flare_compute(c, c->ws.x, c->ws.types, box, pbc, e_out ? c->ws.e : nullptr, f_out ? c->ws.f : nullptr,
                       var_out ? c->ws.var : nullptr);
    if (rc) return rc;
    if (n > 0) {
        if (e_out) FLARE_CUDA(c, cudaMemcpyAsync(e_out, c->ws.e, sizeof(double) * n, cudaMemcpyDeviceToHost, c->stream));
        if (f_out) FLARE_CUDA(c, cudaMemcpyAsync(f_out, c->ws.f, sizeof(double) * 3 * n, cudaMemcpyDeviceToHost, c->stream));
        if (var_out) FLARE_CUDA(c, cudaMemcpyAsync(var_out, c->ws.var, sizeof(double) * n, cudaMemcpyDeviceToHost, c->stream));
    }
    return flare_check(c);
}

static int set_state_impl(flare_ctx* c, const double* pos, const double* vel, const int32_t* types,
                          const double box[9], const int pbc[3], cudaMemcpyKind kind) {
    int rc = need_plain(c, "flare_set_state");
    if (rc) return rc;
    const size_t n = (size_t)c->n;
    if (n > 0 && (!pos || !types)) return fail(c, FLARE_ERR_INVALID_ARG, "pos/types is null");
    FLARE_CUDA(c, cudaSetDevice(c->device));
    rc = setup_grid(c, box, pbc);
    if (rc) return rc;
    if (n > 0) {
        if (pos != c->ws.x) FLARE_CUDA(c, cudaMemcpyAsync(c->ws.x, pos, sizeof(double) * 3 * n, kind, c->stream));
        if (vel) { if (vel != c->ws.v) FLARE_CUDA(c, cudaMemcpyAsync(c->ws.v, vel, sizeof(double) * 3 * n, kind, c->stream)); }
        else FLARE_CUDA(c, cudaMemsetAsync(c->ws.v, 0, sizeof(double) * 3 * n, c->stream));
        if (types != c->ws.types) FLARE_CUDA(c, cudaMemcpyAsync(c->ws.types, types, sizeof(int) * n, kind, c->stream));
    }
    c->state_set = true;
    c->forces_valid = c->var_valid = false;
    return FLARE_OK;
}

int flare_set_state(flare_ctx* c, const double* pos, const double* vel, const int32_t* types, const double box[9],
                    const int pbc[3]) {
    return set_state_impl(c, pos, vel, types, box, pbc, cudaMemcpyDeviceToDevice);
}

int flare_set_state_host(flare_ctx* c, const double* pos, const double* vel, const int32_t* types,
                         const double box[9], const int pbc[3]) {
    return set_state_impl(c, pos, vel, types, box, pbc, cudaMemcpyHostToDevice);
}

static int set_forces_impl(flare_ctx* c, const double* f, cudaMemcpyKind kind) {
    int rc = need_bound(c);
    if (rc) return rc;
    if (!c->state_set) return fail(c, FLARE_ERR_NOT_BOUND, "flare_set_state has not been called");
    if (!f && c->n > 0) return fail(c, FLARE_ERR_INVALID_ARG, "forces pointer is null");
    FLARE_CUDA(c, cudaSetDevice(c->device));
    if (c->n > 0 && f != c->ws.f)
        FLARE_CUDA(c, cudaMemcpyAsync(c->ws.f, f, sizeof(double) * 3 * (size_t)c->n, kind, c->stream));
    c->forces_valid = true;
    return FLARE_OK;
}

int flare_set_forces(flare_ctx* c, const double* f) { return set_forces_impl(c, f, cudaMemcpyDeviceToDevice); }
int flare_set_forces_host(flare_ctx* c, const double* f) { return set_forces_impl(c, f, cudaMemcpyHostToDevice); }

// one velocity-Verlet step (with T_kelvin > 0 bracketed by Nose-Hoover half steps, R19) enqueued through L
static int enqueue_md_step(flare_ctx* c, Launcher& L, double dt_fs, double* var, bool nvt, double gkT, double Q) {
    const int n = (int)c->n;
    Workspace& w = c->ws;
    {
        PhaseScope ps(c, FLARE_PHASE_INTEGRATE);
        if (nvt) run_nh_half(L, w, n, c->d_mass, 0.5 * dt_fs, gkT, Q, w.scal + 12);
        run_kick_drift(L, c->grid, n, w.x, w.v, w.f, w.types, c->d_accel, dt_fs);
    }
    int rc = evaluate(c, L, w.x, w.types, w.e, w.f, var);
    if (rc) return rc;
    {
        PhaseScope ps(c, FLARE_PHASE_INTEGRATE);
        run_kick(L, n, w.v, w.f, w.types, c->d_accel);
        if (nvt) run_nh_half(L, w, n, c->d_mass, 0.5 * dt_fs, gkT, Q, w.scal + 12);
    }
    if (L.err != cudaSuccess) return cuda_fail(c, L.err, L.err_where ? L.err_where : "integrator launch");
    return FLARE_OK;
}

// Small systems are bound by launch latency, not by the GPU (a 256-atom step is ~30 tiny kernels): capture one whole
// MD step -- integrator, neighbour phase with the rebuild chain as a conditional IF node, descriptors, quadratic
// forms, back-propagation, gather -- into a CUDA graph once and replay it ("saturated
// performance ... for small systems").  The launch sequence of a step on a kept candidate list is static, and the
// decision to rebuild is taken on the device, so one graph serves every step of a run.
static bool graph_wanted(const flare_ctx* c) {
    if (c->graph_broken || c->graph_opt == 0 || c->n <= 0) return false;
    if (c->graph_opt == 1) return true;
    // domain mode: every ghost rebuild (each ~10-20 steps) changes the atom count and drops the graph, and a re-capture
    // plus cudaGraphInstantiate costs more than the launch latency saved over so few replays -- plain launches unless asked
    if (c->dom_active) return false;
    return c->n <= 200000;  // automatic: above this a step keeps the GPU busy for longer than its launches take
}

static int capture_md_step(flare_ctx* c, double dt_fs, double* var, bool nvt, double gkT, double Q) {
    if (!c->cap_stream) {
        FLARE_CUDA(c, cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking));
        FLARE_CUDA(c, cudaStreamCreateWithFlags(&c->body_stream, cudaStreamNonBlocking));
    }
    drop_step_graph(c);
    c->plain_stepped = true;  // the caller checked it; dropping the OLD graph must not ask for another plain step
    FLARE_CUDA(c, cudaStreamBeginCapture(c->cap_stream, cudaStreamCaptureModeThreadLocal));
    Launcher L = make_launcher(c);
    L.stream = c->cap_stream;
    L.body_stream = c->body_stream;
    L.capturing = true;
    c->capturing = true;
    const int64_t l0 = c->launches;
    int rc = enqueue_md_step(c, L, dt_fs, var, nvt, gkT, Q);
    c->capturing = false;
    cudaGraph_t g = nullptr;
    cudaError_t e = cudaStreamEndCapture(c->cap_stream, &g);
    c->graph_launches = c->launches - l0;
    c->launches = l0;  // nothing has run yet; replays add their launches
    if (rc == FLARE_OK && e != cudaSuccess) rc = cuda_fail(c, e, "cudaStreamEndCapture");
    if (rc == FLARE_OK) {
        e = cudaGraphInstantiate(&c->step_exec, g, 0);
        if (e != cudaSuccess) rc = cuda_fail(c, e, "cudaGraphInstantiate");
    }
    if (rc != FLARE_OK) {
        if (g) cudaGraphDestroy(g);
        c->step_exec = nullptr;
        cudaGetLastError();
        return rc;
    }
    c->step_graph = g;
    return FLARE_OK;
}

// velocity Verlet; with T_kelvin > 0 each step is bracketed by Nose-Hoover half steps (R19)
static int step_impl(flare_ctx* c, double dt_fs, int n_steps, int want_variance, double T_kelvin, double tau_fs) {
    int rc = need_bound(c);
    if (rc) return rc;
    if (!c->state_set) return fail(c, FLARE_ERR_NOT_BOUND, "flare_set_state has not been called");
    if (n_steps < 0 || !std::isfinite(dt_fs)) return fail(c, FLARE_ERR_INVALID_ARG, "bad dt or n_steps");
    if (want_variance && !c->has_sigma) return fail(c, FLARE_ERR_INVALID_ARG, "variance requested but the model has no sigma");
    FLARE_CUDA(c, cudaSetDevice(c->device));
    const int n = (int)c->n;
    Workspace& w = c->ws;
    double* var = want_variance ? w.var : nullptr;
    Launcher L = make_launcher(c);
    if (!c->forces_valid || (want_variance && !c->var_valid && n_steps == 0)) {
        rc = evaluate(c, L, w.x, w.types, w.e, w.f, var);
        if (rc) return rc;
        c->forces_valid = true;
        c->var_valid = want_variance != 0;
    }
    if (n_steps == 0) return FLARE_OK;
    if (c->accel_dt != dt_fs) {
        // the previous table may still be in flight on the stream: order the overwrite after it
        FLARE_CUDA(c, cudaStreamSynchronize(c->stream));
        for (int s = 0; s < c->bs.S; s++) c->h_accel[s] = 0.5 * dt_fs * kKappa / c->mass[s];
        FLARE_CUDA(c, cudaMemcpyAsync(c->d_accel, c->h_accel.data(), sizeof(double) * kMaxSpecies,
                                      cudaMemcpyHostToDevice, c->stream));
        c->accel_dt = dt_fs;
    }
    const bool nvt = T_kelvin > 0.0;
    const double gkT = (3.0 * (double)n - 3.0) * 8.617333262e-5 * T_kelvin;  // g k_B T, g = 3N - 3 (R13, R19)
    const double Q = gkT * tau_fs * tau_fs;
    flare_ctx::StepKey key;
    key.dt = dt_fs; key.T = nvt ? T_kelvin : 0.0; key.tau = nvt ? tau_fs : 0.0; key.var = want_variance ? 1 : 0;
    for (int step = 0; step < n_steps; step++) {
        // a step can be replayed from the graph when its launch sequence is the captured one: the candidate list is
        // kept (or there is none), and a plain step with the same parameters has run (every kernel is loaded)
        const bool static_chain = eff_skin(c) == 0.0 || c->list_valid;
        if (graph_wanted(c) && static_chain && c->plain_stepped && c->plain_key == key) {
            if (!c->step_exec || !(c->graph_key == key)) {
                rc = capture_md_step(c, dt_fs, var, nvt, gkT, Q);
                if (rc != FLARE_OK) { c->graph_broken = true; c->step_exec = nullptr; }
                else c->graph_key = key;
            }
            if (c->step_exec) {
                FLARE_CUDA(c, cudaGraphLaunch(c->step_exec, c->stream));
                c->launches += c->graph_launches;
                c->graph_replays++;
                continue;
            }
        }
        rc = enqueue_md_step(c, L, dt_fs, var, nvt, gkT, Q);
        if (rc) return rc;
        c->plain_stepped = true;
        c->plain_key = key;
    }
    c->var_valid = want_variance != 0;
    return FLARE_OK;
}

int flare_step(flare_ctx* c, double dt_fs, int n_steps, int want_variance) {
    return step_impl(c, dt_fs, n_steps, want_variance, 0.0, 0.0);
}

int flare_step_nvt(flare_ctx* c, double dt_fs, int n_steps, int want_variance, double T_kelvin, double tau_fs) {
    if (!c) return FLARE_ERR_INVALID_ARG;
    if (!(T_kelvin > 0.0) || !(tau_fs > 0.0) || !std::isfinite(T_kelvin) || !std::isfinite(tau_fs))
        return fail(c, FLARE_ERR_INVALID_ARG, "thermostat temperature and time constant must be > 0");
    if (c->n >= 0 && c->n < 2) return fail(c, FLARE_ERR_INVALID_ARG, "the thermostat needs at least 2 atoms (g = 3N - 3)");
    return step_impl(c, dt_fs, n_steps, want_variance, T_kelvin, tau_fs);
}

// ---------------------------------------------------------------- multi-GPU domain decomposition (domain.cu)
static int need_domain(flare_ctx* c) {
    int rc = need_bound(c);
    if (rc) return rc;
    if (!c->dom_active) return fail(c, FLARE_ERR_NOT_BOUND, "flare_domain_begin has not been called");
    return FLARE_OK;
}

int flare_domain_begin(flare_ctx* c, int64_t n_owned, const double* pos, const double* vel, const int32_t* types,
                       const int64_t* tags, const double box[9], const int pbc[3], double trigger_displacement) {
    int rc = need_bound(c);
    if (rc) return rc;
    if (n_owned < 0 || n_owned > c->n_cap) return fail(c, FLARE_ERR_WORKSPACE_TOO_SMALL, "n_owned exceeds the bound capacity");
    if (n_owned > 0 && (!pos || !types || !tags)) return fail(c, FLARE_ERR_INVALID_ARG, "pos/types/tags is null");
    if (!(trigger_displacement >= 0.0)) return fail(c, FLARE_ERR_INVALID_ARG, "trigger displacement must be >= 0");
    FLARE_CUDA(c, cudaSetDevice(c->device));
    rc = setup_grid(c, box, pbc);
    if (rc) return rc;  // the context is left as it was
    c->n = n_owned;
    const size_t n = (size_t)n_owned;
    if (n > 0) {
        FLARE_CUDA(c, cudaMemcpyAsync(c->ws.x, pos, sizeof(double) * 3 * n, cudaMemcpyDeviceToDevice, c->stream));
        if (vel) FLARE_CUDA(c, cudaMemcpyAsync(c->ws.v, vel, sizeof(double) * 3 * n, cudaMemcpyDeviceToDevice, c->stream));
        else FLARE_CUDA(c, cudaMemsetAsync(c->ws.v, 0, sizeof(double) * 3 * n, c->stream));
        FLARE_CUDA(c, cudaMemsetAsync(c->ws.f, 0, sizeof(double) * 3 * n, c->stream));
        FLARE_CUDA(c, cudaMemcpyAsync(c->ws.types, types, sizeof(int) * n, cudaMemcpyDeviceToDevice, c->stream));
        FLARE_CUDA(c, cudaMemcpyAsync(c->ws.tag, tags, sizeof(long long) * n, cudaMemcpyDeviceToDevice, c->stream));
    }
    int h[kDomInts] = {0};
    h[kDomNLocal] = h[kDomNOwned] = (int)n_owned;
    FLARE_CUDA(c, cudaStreamSynchronize(c->stream));
    FLARE_CUDA(c, cudaMemcpy(c->ws.dom, h, sizeof(h), cudaMemcpyHostToDevice));
    c->dom_active = true;
    c->dom_trigger = trigger_displacement;
    c->dom_limit = 0.0;
    c->dom_n_owned = n_owned;
    for (int q = 0; q < 4; q++) c->dom_send[q] = c->dom_recv_cnt[q] = c->dom_recv_off[q] = 0;
    c->state_set = true;
    c->forces_valid = c->var_valid = false;
    c->list_valid = false;
    c->pairf_valid = false;
    drop_step_graph(c);
    return FLARE_OK;
}

int flare_domain_migrate_pack(flare_ctx* c, int axis, double lo_bound, double hi_bound, double shift_lo,
                              double shift_hi, double* msg_lo, double* msg_hi, int64_t cap_rows) {
    int rc = need_domain(c);
    if (rc) return rc;
    if (axis < 0 || axis > 2 || !msg_lo || !msg_hi || cap_rows < 0 || cap_rows > 0x7fffffff / kDomFullRow)
        return fail(c, FLARE_ERR_INVALID_ARG, "bad axis, message pointer or capacity");
    FLARE_CUDA(c, cudaSetDevice(c->device));
    Launcher L = make_launcher(c);
    const int nb = (int)c->n_cap;
    dom_set_counts(L, c->ws, kDomNOwned, true, false);  // ghosts are dropped: the local set is the owned set
    const double inf = HUGE_VAL;
    const DomSel s{axis, kDomNOwned, -inf, lo_bound, hi_bound, inf};
    int* leave_lo = c->ws.rank_in_cell;                // scratch (free between evaluations)
    int* leave_hi = c->ws.rank_in_cell + (nb + 1) / 2;
    int* stay = c->ws.cell_of;
    dom_select(L, c->ws, s, nb, leave_lo, leave_hi, stay, std::max(nb / 2, 1));
    dom_commit_lists(L, c->ws, kDomMig, kDomMig + 1, std::max(nb / 2, 1));
    double sh[3] = {0.0, 0.0, 0.0};
    sh[axis] = shift_lo;
    dom_pack_full(L, c->ws, leave_lo, kDomMig, sh, true, msg_lo, (int)cap_rows);
    sh[axis] = shift_hi;
    dom_pack_full(L, c->ws, leave_hi, kDomMig + 1, sh, true, msg_hi, (int)cap_rows);
    dom_compact_stay(L, c->ws, stay, nb);
    if (L.err != cudaSuccess) return cuda_fail(c, L.err, L.err_where ? L.err_where : "domain launch");
    c->list_valid = false;
    c->pairf_valid = false;
    return FLARE_OK;
}

int flare_domain_migrate_unpack(flare_ctx* c, const double* msg_lo_in, const double* msg_hi_in, int64_t cap_rows) {
    int rc = need_domain(c);
    if (rc) return rc;
    if (cap_rows < 0 || cap_rows > 0x7fffffff / kDomFullRow) return fail(c, FLARE_ERR_INVALID_ARG, "bad message capacity");
    FLARE_CUDA(c, cudaSetDevice(c->device));
    Launcher L = make_launcher(c);
    if (msg_lo_in) dom_append(L, c->ws, msg_lo_in, (int)c->n_cap, (int)cap_rows, -1, true);
    if (msg_hi_in) dom_append(L, c->ws, msg_hi_in, (int)c->n_cap, (int)cap_rows, -1, true);
    if (L.err != cudaSuccess) return cuda_fail(c, L.err, L.err_where ? L.err_where : "domain launch");
    return FLARE_OK;
}

int flare_domain_border_pack(flare_ctx* c, int phase, int axis, double lo_a, double lo_b, double hi_a, double hi_b,
                             double shift_lo, double shift_hi, double* msg_lo, double* msg_hi, int64_t cap_rows) {
    int rc = need_domain(c);
    if (rc) return rc;
    if (phase < 0 || phase > 1 || axis < 0 || axis > 2 || !msg_lo || !msg_hi || cap_rows < 0 ||
        cap_rows > 0x7fffffff / kDomFullRow)
        return fail(c, FLARE_ERR_INVALID_ARG, "bad phase, axis, message pointer or capacity");
    FLARE_CUDA(c, cudaSetDevice(c->device));
    Launcher L = make_launcher(c);
    if (phase == 0) dom_set_counts(L, c->ws, kDomNOwned, true, false);  // a new ghost shell starts after the owned atoms
    const DomSel s{axis, kDomNLocal, lo_a, lo_b, hi_a, hi_b};
    int* list_lo = c->ws.send_idx + (size_t)(2 * phase) * c->dom_list_cap;
    int* list_hi = c->ws.send_idx + (size_t)(2 * phase + 1) * c->dom_list_cap;
    dom_select(L, c->ws, s, (int)c->n_cap, list_lo, list_hi, nullptr, c->dom_list_cap);
    dom_commit_lists(L, c->ws, kDomSend + 2 * phase, kDomSend + 2 * phase + 1, c->dom_list_cap);
    for (int side = 0; side < 2; side++) {
        double* sh = c->dom_shift[2 * phase + side];
        sh[0] = sh[1] = sh[2] = 0.0;
        sh[axis] = side == 0 ? shift_lo : shift_hi;
        dom_pack_full(L, c->ws, side == 0 ? list_lo : list_hi, kDomSend + 2 * phase + side, sh, c->forces_valid,
                      side == 0 ? msg_lo : msg_hi, (int)cap_rows);
    }
    if (L.err != cudaSuccess) return cuda_fail(c, L.err, L.err_where ? L.err_where : "domain launch");
    return FLARE_OK;
}

int flare_domain_border_unpack(flare_ctx* c, int phase, const double* msg_lo_in, const double* msg_hi_in,
                               int64_t cap_rows) {
    int rc = need_domain(c);
    if (rc) return rc;
    if (phase < 0 || phase > 1 || cap_rows < 0 || cap_rows > 0x7fffffff / kDomFullRow)
        return fail(c, FLARE_ERR_INVALID_ARG, "bad phase or message capacity");
    FLARE_CUDA(c, cudaSetDevice(c->device));
    Launcher L = make_launcher(c);
    // an absent neighbour (null) still records an empty ghost block
    double* d_empty = c->ws.red;  // 8 doubles of reduction scratch
    if (!msg_lo_in || !msg_hi_in) FLARE_CUDA(c, cudaMemsetAsync(d_empty, 0, sizeof(double) * kDomHeader, c->stream));
    dom_append(L, c->ws, msg_lo_in ? msg_lo_in : d_empty, (int)c->n_cap, (int)cap_rows, 2 * phase, false);
    dom_append(L, c->ws, msg_hi_in ? msg_hi_in : d_empty, (int)c->n_cap, (int)cap_rows, 2 * phase + 1, false);
    if (L.err != cudaSuccess) return cuda_fail(c, L.err, L.err_where ? L.err_where : "domain launch");
    return FLARE_OK;
}

int flare_domain_commit(flare_ctx* c, int64_t counts[14]) {
    int rc = need_domain(c);
    if (rc) return rc;
    FLARE_CUDA(c, cudaSetDevice(c->device));
    FLARE_CUDA(c, cudaStreamSynchronize(c->stream));
    int h[kDomInts];
    FLARE_CUDA(c, cudaMemcpy(h, c->ws.dom, sizeof(h), cudaMemcpyDeviceToHost));
    rc = flare_check(c);  // message / list / capacity overflow of the rebuild
    if (rc) return rc;
    c->n = h[kDomNLocal];
    c->dom_n_owned = h[kDomNOwned];
    for (int q = 0; q < 4; q++) {
        c->dom_send[q] = h[kDomSend + q];
        c->dom_recv_cnt[q] = h[kDomRecvCnt + q];
        c->dom_recv_off[q] = h[kDomRecvOff + q];
    }
    FLARE_CUDA(c, cudaMemsetAsync(c->ws.dom + kDomNeed, 0, sizeof(int), c->stream));
    if (c->n > 0)  // displacements are measured from here on
        FLARE_CUDA(c, cudaMemcpyAsync(c->ws.dom_ref, c->ws.x, sizeof(double) * 3 * (size_t)c->n, cudaMemcpyDeviceToDevice, c->stream));
    c->list_valid = false;  // membership changed: the candidate list is rebuilt by the next evaluation
    c->pairf_valid = false;
    drop_step_graph(c);
    if (counts) {
        counts[0] = h[kDomNLocal];
        counts[1] = h[kDomNOwned];
        for (int q = 0; q < 4; q++) {
            counts[2 + q] = h[kDomSend + q];
            counts[6 + q] = h[kDomRecvCnt + q];
            counts[10 + q] = h[kDomRecvOff + q];
        }
    }
    return FLARE_OK;
}

int flare_domain_forward_pack(flare_ctx* c, int phase, double* msg_lo, double* msg_hi) {
    int rc = need_domain(c);
    if (rc) return rc;
    if (phase < 0 || phase > 1 || !msg_lo || !msg_hi) return fail(c, FLARE_ERR_INVALID_ARG, "bad phase or message pointer");
    FLARE_CUDA(c, cudaSetDevice(c->device));
    Launcher L = make_launcher(c);
    for (int side = 0; side < 2; side++) {
        const int q = 2 * phase + side;
        dom_pack_fwd(L, c->ws, c->ws.send_idx + (size_t)q * c->dom_list_cap, c->dom_send[q], c->dom_shift[q],
                     side == 0 ? msg_lo : msg_hi);
    }
    if (L.err != cudaSuccess) return cuda_fail(c, L.err, L.err_where ? L.err_where : "domain launch");
    return FLARE_OK;
}

int flare_domain_forward_unpack(flare_ctx* c, int phase, const double* msg_lo_in, const double* msg_hi_in) {
    int rc = need_domain(c);
    if (rc) return rc;
    if (phase < 0 || phase > 1) return fail(c, FLARE_ERR_INVALID_ARG, "bad phase");
    FLARE_CUDA(c, cudaSetDevice(c->device));
    Launcher L = make_launcher(c);
    if (msg_lo_in) dom_unpack_fwd(L, c->ws, msg_lo_in, c->dom_recv_off[2 * phase], c->dom_recv_cnt[2 * phase]);
    if (msg_hi_in) dom_unpack_fwd(L, c->ws, msg_hi_in, c->dom_recv_off[2 * phase + 1], c->dom_recv_cnt[2 * phase + 1]);
    if (L.err != cudaSuccess) return cuda_fail(c, L.err, L.err_where ? L.err_where : "domain launch");
    return FLARE_OK;
}

int flare_domain_signal(flare_ctx* c, int32_t* flag_out) {
    int rc = need_domain(c);
    if (rc) return rc;
    if (!flag_out) return fail(c, FLARE_ERR_INVALID_ARG, "flag pointer is null");
    FLARE_CUDA(c, cudaSetDevice(c->device));
    if (eff_skin(c) > 0.0 && c->dom_trigger > 0.0)
        FLARE_CUDA(c, cudaMemcpyAsync(flag_out, c->ws.dom + kDomNeed, sizeof(int), cudaMemcpyDeviceToDevice, c->stream));
    else
        FLARE_CUDA(c, cudaMemsetAsync(flag_out, 1, 1, c->stream));  // no candidate list, no displacement tracking: always
    return FLARE_OK;
}

int flare_domain_status(flare_ctx* c, int32_t* status_out) {
    int rc = need_domain(c);
    if (rc) return rc;
    if (!status_out) return fail(c, FLARE_ERR_INVALID_ARG, "status pointer is null");
    FLARE_CUDA(c, cudaSetDevice(c->device));
    FLARE_CUDA(c, cudaMemcpyAsync(status_out, c->ws.flags, sizeof(int), cudaMemcpyDeviceToDevice, c->stream));
    return FLARE_OK;
}

int flare_domain_set_limit(flare_ctx* c, double max_displacement) {
    int rc = need_domain(c);
    if (rc) return rc;
    if (!(max_displacement >= 0.0)) return fail(c, FLARE_ERR_INVALID_ARG, "the displacement limit must be >= 0");
    if (max_displacement > 0.0 && c->dom_trigger > 0.0 && !(max_displacement > c->dom_trigger))
        return fail(c, FLARE_ERR_INVALID_ARG, "the displacement limit must exceed the trigger displacement of flare_domain_begin");
    if (max_displacement != c->dom_limit) drop_step_graph(c);  // a captured step has the old limit baked in
    c->dom_limit = max_displacement;
    return FLARE_OK;
}

int flare_domain_get_tags(flare_ctx* c, int64_t* tags_out) {
    int rc = need_domain(c);
    if (rc) return rc;
    if (!tags_out && c->n > 0) return fail(c, FLARE_ERR_INVALID_ARG, "tags pointer is null");
    FLARE_CUDA(c, cudaSetDevice(c->device));
    if (c->n > 0)
        FLARE_CUDA(c, cudaMemcpyAsync(tags_out, c->ws.tag, sizeof(long long) * (size_t)c->n, cudaMemcpyDeviceToDevice, c->stream));
    return FLARE_OK;
}

int flare_get_thermostat(flare_ctx* c, double* xi, double* eta) {
    int rc = need_bound(c);
    if (rc) return rc;
    FLARE_CUDA(c, cudaSetDevice(c->device));
    FLARE_CUDA(c, cudaStreamSynchronize(c->stream));
    double h[2] = {0.0, 0.0};
    FLARE_CUDA(c, cudaMemcpy(h, c->ws.scal + 12, sizeof(h), cudaMemcpyDeviceToHost));
    if (xi) *xi = h[0];
    if (eta) *eta = h[1];
    return FLARE_OK;
}

int flare_set_thermostat(flare_ctx* c, double xi, double eta) {
    int rc = need_bound(c);
    if (rc) return rc;
    if (!std::isfinite(xi) || !std::isfinite(eta)) return fail(c, FLARE_ERR_INVALID_ARG, "non-finite thermostat state");
    FLARE_CUDA(c, cudaSetDevice(c->device));
    FLARE_CUDA(c, cudaStreamSynchronize(c->stream));
    const double h[2] = {xi, eta};
    FLARE_CUDA(c, cudaMemcpy(c->ws.scal + 12, h, sizeof(h), cudaMemcpyHostToDevice));
    return FLARE_OK;
}

int flare_get_virial(flare_ctx* c, double virial[9]) {
    int rc = need_bound(c);
    if (rc) return rc;
    if (!virial) return fail(c, FLARE_ERR_INVALID_ARG, "virial is null");
    if (!c->pairf_valid) return fail(c, FLARE_ERR_NOT_BOUND, "no evaluation has been run");
    FLARE_CUDA(c, cudaSetDevice(c->device));
    for (int q = 0; q < 9; q++) virial[q] = 0.0;
    if (c->n == 0) return FLARE_OK;
    Launcher L = make_launcher(c);
    run_virial(L, c->grid, c->ws, (int)c->n, c->mmax, c->ws.scal);
    if (L.err != cudaSuccess) return cuda_fail(c, L.err, "virial launch");
    FLARE_CUDA(c, cudaMemcpyAsync(virial, c->ws.scal, sizeof(double) * 9, cudaMemcpyDeviceToHost, c->stream));
    return flare_check(c);
}

int flare_virial_static(flare_ctx* c, double* virial_dev) {
    int rc = need_bound(c);
    if (rc) return rc;
    if (!virial_dev) return fail(c, FLARE_ERR_INVALID_ARG, "virial_dev is null");
    static_assert(FLARE_VIRIAL_STATIC_MAX_ATOMS == flare::kVirialStaticMaxAtoms, "header constant out of step");
    if (c->n > (int64_t)FLARE_VIRIAL_STATIC_MAX_ATOMS)
        return fail(c, FLARE_ERR_INVALID_ARG,
                    "flare_virial_static: " + std::to_string(c->n) + " atoms exceed the static scratch array's limit of " +
                        std::to_string((int64_t)FLARE_VIRIAL_STATIC_MAX_ATOMS) + " atoms; use flare_get_virial");
    if (!c->pairf_valid) return fail(c, FLARE_ERR_NOT_BOUND, "no evaluation has been run");
    FLARE_CUDA(c, cudaSetDevice(c->device));
    Launcher L = make_launcher(c);
    const cudaError_t e = run_virial_static(L, c->device, c->grid, c->ws, (int)c->n, c->mmax, virial_dev);
    if (e != cudaSuccess) return cuda_fail(c, e, L.err_where ? L.err_where : "flare_virial_static");
    return FLARE_OK;
}

int flare_analyze(flare_ctx* c, double unc_threshold, int species_a, int species_b, double r_coord, double* max_unc,
                  int64_t* n_above, int32_t* coord, int64_t* coord_hist) {
    int rc = need_bound(c);
    if (rc) return rc;
    if (!c->pairf_valid) return fail(c, FLARE_ERR_NOT_BOUND, "no evaluation has been run");
    const bool want_unc = max_unc || n_above;
    const bool want_coord = coord || coord_hist;
    if (want_unc && !c->last_eval_var) return fail(c, FLARE_ERR_INVALID_ARG, "the last evaluation had no variances");
    if (want_coord) {
        if (species_a < 0 || species_a >= c->bs.S || species_b < 0 || species_b >= c->bs.S)
            return fail(c, FLARE_ERR_INVALID_ARG, "species out of range");
        // the neighbour list only holds pairs inside r_cut[a][b]
        if (!(r_coord > 0.0) || r_coord > c->bs.rc[species_a * c->bs.S + species_b])
            return fail(c, FLARE_ERR_INVALID_ARG, "r_coord must be in (0, r_cut[a][b]]");
    }
    FLARE_CUDA(c, cudaSetDevice(c->device));
    unsigned long long h[18] = {0};
    if (c->n > 0 && (want_unc || want_coord)) {
        Launcher L = make_launcher(c);
        run_analyze(L, c->grid, c->ws, (int)c->n, c->mmax, want_unc, unc_threshold, species_a, species_b, r_coord,
                    want_coord, coord, c->ws.ascal);
        if (L.err != cudaSuccess) return cuda_fail(c, L.err, "analysis launch");
        FLARE_CUDA(c, cudaMemcpyAsync(h, c->ws.ascal, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    }
    rc = flare_check(c);
    if (rc) return rc;
    if (max_unc) { double u; memcpy(&u, &h[0], sizeof(u)); *max_unc = u; }
    if (n_above) *n_above = (int64_t)h[1];
    if (coord_hist) for (int q = 0; q < 16; q++) coord_hist[q] = (int64_t)h[2 + q];
    return FLARE_OK;
}

static int get_state_impl(flare_ctx* c, double* pos, double* vel, double* e, double* f, double* var,
                          cudaMemcpyKind kind) {
    int rc = need_bound(c);
    if (rc) return rc;
    if (!c->state_set) return fail(c, FLARE_ERR_NOT_BOUND, "flare_set_state has not been called");
    if (var && !c->var_valid) return fail(c, FLARE_ERR_INVALID_ARG, "variances were not evaluated");
    if ((e || f) && !c->forces_valid) return fail(c, FLARE_ERR_INVALID_ARG, "forces were not evaluated yet");
    const size_t n = (size_t)c->n;
    if (n == 0) return FLARE_OK;
    FLARE_CUDA(c, cudaSetDevice(c->device));
    if (pos) FLARE_CUDA(c, cudaMemcpyAsync(pos, c->ws.x, sizeof(double) * 3 * n, kind, c->stream));
    if (vel) FLARE_CUDA(c, cudaMemcpyAsync(vel, c->ws.v, sizeof(double) * 3 * n, kind, c->stream));
    if (e) FLARE_CUDA(c, cudaMemcpyAsync(e, c->ws.e, sizeof(double) * n, kind, c->stream));
    if (f) FLARE_CUDA(c, cudaMemcpyAsync(f, c->ws.f, sizeof(double) * 3 * n, kind, c->stream));
    if (var) FLARE_CUDA(c, cudaMemcpyAsync(var, c->ws.var, sizeof(double) * n, kind, c->stream));
    return FLARE_OK;
}

int flare_get_state(flare_ctx* c, double* pos, double* vel, double* e, double* f, double* var) {
    return get_state_impl(c, pos, vel, e, f, var, cudaMemcpyDeviceToDevice);
}

int flare_get_state_host(flare_ctx* c, double* pos, double* vel, double* e, double* f, double* var) {
    int rc = get_state_impl(c, pos, vel, e, f, var, cudaMemcpyDeviceToHost);
    if (rc) return rc;
    return flare_check(c);
}

int flare_get_neighbors(flare_ctx* c, int32_t* cnt, int32_t* idx, int32_t stride) {
    int rc = need_bound(c);
    if (rc) return rc;
    if (!c->have_grid) return fail(c, FLARE_ERR_NOT_BOUND, "no evaluation has been run");
    if (!cnt || !idx || stride < 1) return fail(c, FLARE_ERR_INVALID_ARG, "bad output arrays");
    rc = flare_check(c);
    if (rc) return rc;
    const size_t n = (size_t)c->n;
    if (n == 0) return FLARE_OK;
    std::vector<int> h_cnt(n), h_idx(n * c->mmax);
    std::vector<AtomS> h_atoms(n);
    FLARE_CUDA(c, cudaMemcpy(h_cnt.data(), c->ws.nbr_cnt, sizeof(int) * n, cudaMemcpyDeviceToHost));
    FLARE_CUDA(c, cudaMemcpy(h_idx.data(), c->ws.nbr_idx, sizeof(int) * n * c->mmax, cudaMemcpyDeviceToHost));
    FLARE_CUDA(c, cudaMemcpy(h_atoms.data(), c->ws.atoms, sizeof(AtomS) * n, cudaMemcpyDeviceToHost));
    std::vector<int> row;
    int status = FLARE_OK;
    for (size_t k = 0; k < n; k++) {
        const int i = h_atoms[k].orig;
        row.clear();
        for (int s = 0; s < h_cnt[k]; s++) row.push_back(h_atoms[h_idx[k * c->mmax + s]].orig);
        std::sort(row.begin(), row.end());
        cnt[i] = h_cnt[k];
        for (int s = 0; s < stride; s++) idx[(size_t)i * stride + s] = s < (int)row.size() ? row[s] : -1;
        if ((int)row.size() > stride) status = FLARE_ERR_INVALID_ARG;
    }
    if (status) return fail(c, status, "stride smaller than a neighbour count");
    return FLARE_OK;
}

int flare_get_descriptors(flare_ctx* c, double* bhat, double* nrm) {
    int rc = need_bound(c);
    if (rc) return rc;
    if (!c->have_grid) return fail(c, FLARE_ERR_NOT_BOUND, "no evaluation has been run");
    if (!bhat || !nrm) return fail(c, FLARE_ERR_INVALID_ARG, "bad output arrays");
    rc = flare_check(c);
    if (rc) return rc;
    const int n = (int)c->n;
    const int P = c->bs.P;
    std::vector<AtomS> h_atoms((size_t)n);
    std::vector<int> h_aor((size_t)n);
    std::vector<unsigned char> h_gid((size_t)n);
    if (n == 0) return FLARE_OK;
    FLARE_CUDA(c, cudaMemcpy(h_atoms.data(), c->ws.atoms, sizeof(AtomS) * n, cudaMemcpyDeviceToHost));
    FLARE_CUDA(c, cudaMemcpy(h_aor.data(), c->ws.atom_of_row, sizeof(int) * n, cudaMemcpyDeviceToHost));
    FLARE_CUDA(c, cudaMemcpy(h_gid.data(), c->ws.gid, n, cudaMemcpyDeviceToHost));
    const auto& comps = c->sets[c->sparse].comps;
    Launcher L = make_launcher(c);
    std::vector<double> hb, hn;
    for (int row0 = 0; row0 < n; row0 += c->chunk_cap) {
        const int nrows = std::min(c->chunk_cap, n - row0);
        run_descriptors(L, c->grid, c->bs, c->yn, c->ws, c->mmax, c->groups.data(), c->n_groups, row0, nrows, c->ws.Bh,
                        c->ld, c->ws.nrm, false);
        if (L.err != cudaSuccess) return cuda_fail(c, L.err, "descriptor launch");
        hb.resize((size_t)nrows * c->ld);
        hn.resize(nrows);
        FLARE_CUDA(c, cudaMemcpyAsync(hb.data(), c->ws.Bh, sizeof(double) * hb.size(), cudaMemcpyDeviceToHost, c->stream));
        FLARE_CUDA(c, cudaMemcpyAsync(hn.data(), c->ws.nrm, sizeof(double) * nrows, cudaMemcpyDeviceToHost, c->stream));
        FLARE_CUDA(c, cudaStreamSynchronize(c->stream));
        for (int r = 0; r < nrows; r++) {
            const int k = h_aor[row0 + r];
            const int i = h_atoms[k].orig;
            const std::vector<int>& comp = comps[h_gid[k]];  // compacted -> dense component (identity in dense mode)
            double* dst = bhat + (size_t)i * P;
            for (int p = 0; p < P; p++) dst[p] = 0.0;
            // rows hold the unnormalised B; atoms without neighbours (empty group) have no row content at all (R8)
            const double nr = comp.empty() ? 0.0 : std::sqrt(hn[r]);  // the workspace holds ||B||^2
            const double inv = nr > 0.0 ? 1.0 / nr : 0.0;
            for (size_t q = 0; q < comp.size(); q++) dst[comp[q]] = hb[(size_t)r * c->ld + q] * inv;
            nrm[i] = nr;
        }
    }
    return FLARE_OK;
}

int flare_get_groups(flare_ctx* c, int32_t* n_groups, int64_t* rows, int32_t* comps) {
    int rc = need_bound(c);
    if (rc) return rc;
    if (!c->have_grid) return fail(c, FLARE_ERR_NOT_BOUND, "no evaluation has been run");
    if (!n_groups || !rows || !comps) return fail(c, FLARE_ERR_INVALID_ARG, "bad output arrays");
    rc = flare_check(c);
    if (rc) return rc;
    std::vector<int> start(c->n_groups + 1, 0);
    if (c->n > 0)
        FLARE_CUDA(c, cudaMemcpy(start.data(), c->ws.group_start, sizeof(int) * (c->n_groups + 1), cudaMemcpyDeviceToHost));
    *n_groups = c->n_groups;
    for (int g = 0; g < c->n_groups; g++) {
        rows[g] = start[g + 1] - start[g];
        comps[g] = c->groups[g].P;
    }
    return FLARE_OK;
}

int flare_get_rows(flare_ctx* c, int32_t* row) {
    int rc = need_bound(c);
    if (rc) return rc;
    if (!c->have_grid) return fail(c, FLARE_ERR_NOT_BOUND, "no evaluation has been run");
    if (!row) return fail(c, FLARE_ERR_INVALID_ARG, "bad output array");
    rc = flare_check(c);
    if (rc) return rc;
    const size_t n = (size_t)c->n;
    if (n == 0) return FLARE_OK;
    std::vector<AtomS> h_atoms(n);
    std::vector<int> h_row(n);
    FLARE_CUDA(c, cudaMemcpy(h_atoms.data(), c->ws.atoms, sizeof(AtomS) * n, cudaMemcpyDeviceToHost));
    FLARE_CUDA(c, cudaMemcpy(h_row.data(), c->ws.row_of, sizeof(int) * n, cudaMemcpyDeviceToHost));
    for (size_t k = 0; k < n; k++) row[h_atoms[k].orig] = h_row[k];
    return FLARE_OK;
}

int flare_get_timings(flare_ctx* c, double* ms, int64_t* launches) {
    if (!c || !ms) return FLARE_ERR_INVALID_ARG;
    FLARE_CUDA(c, cudaStreamSynchronize(c->stream));
    for (int p = 0; p < FLARE_N_PHASES; p++) {
        PhaseEvents& pe = c->phases[p];
        double tot = 0.0;
        for (size_t i = 0; i < pe.used; i++) {
            float t = 0.f;
            if (cudaEventElapsedTime(&t, pe.start[i], pe.stop[i]) == cudaSuccess) tot += t;
        }
        ms[p] = tot;
        if (launches) launches[p] = pe.launches;
        pe.used = 0;
        pe.launches = 0;
    }
    return FLARE_OK;
}

int64_t flare_kernel_launches(const flare_ctx* c) { return c ? c->launches : 0; }

const char* flare_last_error(const flare_ctx* c) { return c ? c->err.c_str() : "null context"; }

#pragma GCC visibility pop
}  // extern "C"
