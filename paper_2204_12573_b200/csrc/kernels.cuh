// kernels.cuh -- host-side launch plumbing shared by the translation units of libflare_b200.so:
// the workspace layout, the stream/launch-count/timing wrapper, and the per-stage entry points.
#pragma once
#include <utility>
#include <vector>

#include "basis.cuh"
#include "common.cuh"

namespace flare {

constexpr int kMaxGroups = 64;  // quadratic-form groups: (central species) or (species, neighbour mask)
constexpr int kNumPhases = 6;
constexpr int kSkinStride = 64;  // row stride of the skin (candidate) list: one 64-bit hit mask per atom

// ---- domain decomposition (domain.cu): device-side counters Workspace::dom[] and message layout
constexpr int kDomNLocal = 0;   // atoms in the state arrays: owned + ghosts appended so far
constexpr int kDomNOwned = 1;   // owned atoms (the first ones)
constexpr int kDomSend = 2;     // [4] entries of the send lists x-lo, x-hi, y-lo, y-hi
constexpr int kDomRecvCnt = 6;  // [4] ghosts received from x-lo, x-hi, y-lo, y-hi
constexpr int kDomRecvOff = 10; // [4] first slot of each of those ghost blocks
constexpr int kDomNeed = 15;    // non-zero: an atom has moved further than the halo skin allows since the last rebuild
constexpr int kDomTot = 16;     // [3] totals of the running selection (lo, hi, stay)
constexpr int kDomMig = 20;     // [2] atoms leaving through the lo / hi face of the running migration phase
constexpr int kDomInts = 32;
constexpr int kDomHeader = 8;   // doubles before the first row of a message ([0] = row count)
constexpr int kDomFullRow = 11; // x, v, f, type, tag
constexpr int kDomFwdRow = 9;   // x, v, f

// selection along one axis: bit 0 = coordinate in [lo_a, lo_b), bit 1 = in [hi_a, hi_b); over the first dom[n_from] atoms
struct DomSel {
    int axis, n_from;
    double lo_a, lo_b, hi_a, hi_b;
};

// Per-context launch state: the dynamic shared-memory limit a kernel has been configured for and its occupancy.
// cudaFuncSetAttribute acts on the CURRENT device only, so this lives in the context (one context = one device),
// not in function-local statics: a second context on another GPU of the same process configures its own copy.
struct LaunchCache {
    struct Entry { const void* fn; size_t smem; int occ; };
    std::vector<Entry> entries;
    Entry& find(const void* fn) {
        for (Entry& e : entries) if (e.fn == fn) return e;
        entries.push_back(Entry{fn, 0, 0});
        return entries.back();
    }
};

// Launch wrapper: all kernels go to one stream; counts launches; keeps the first CUDA error.
struct Launcher {
    cudaStream_t stream = nullptr;
    int64_t* launch_count = nullptr;
    LaunchCache* cache = nullptr;
    cudaError_t err = cudaSuccess;
    const char* err_where = nullptr;

    void fail_here(cudaError_t e, const char* where) {
        if (e != cudaSuccess && err == cudaSuccess) { err = e; err_where = where; }
    }

    // raise the kernel's dynamic shared-memory limit (needed above 48 KB) once per context and size
    template <class... KArgs>
    void ensure_smem(void (*kernel)(KArgs...), size_t bytes) {
        if (bytes <= 48 * 1024 || err != cudaSuccess) return;
        LaunchCache::Entry local{nullptr, 0, 0};
        LaunchCache::Entry& e = cache ? cache->find(reinterpret_cast<const void*>(kernel)) : local;
        if (bytes <= e.smem) return;
        cudaError_t rc = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
        if (rc != cudaSuccess) { err = rc; err_where = "cudaFuncSetAttribute(MaxDynamicSharedMemorySize)"; return; }
        e.smem = bytes;
    }
    // resident CTAs per SM of a kernel at this block size / shared memory (queried once per context)
    template <class... KArgs>
    int occupancy(void (*kernel)(KArgs...), int threads, size_t smem, int fallback) {
        LaunchCache::Entry local{nullptr, 0, 0};
        LaunchCache::Entry& e = cache ? cache->find(reinterpret_cast<const void*>(kernel)) : local;
        if (e.occ == 0) {
            int occ = 0;
            if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel, threads, smem) != cudaSuccess || occ < 1)
                occ = fallback;
            e.occ = occ;
        }
        return e.occ;
    }

    template <class... KArgs, class... Args>
    void launch(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, Args&&... args) {
        if (grid.x == 0 || grid.y == 0 || grid.z == 0 || err != cudaSuccess) return;
        kernel<<<grid, block, smem, stream>>>(std::forward<Args>(args)...);
        // kernels captured into a conditional IF body run only when the device switches the node on: not counted
        if (launch_count && outer_stream == nullptr) ++*launch_count;
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess && err == cudaSuccess) { err = e; err_where = "kernel launch"; }
    }
    // ---- side stream: the per-group launches of a phase are independent (disjoint rows), so the groups with few rows
    // run beside the large one instead of after it (their kernels cannot fill the GPU by themselves)
    cudaStream_t side = nullptr;
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
    int big_group = -1;  // group expected to hold most rows (a scheduling hint only); -1: no overlap
    cudaStream_t main_stream = nullptr;
    bool forked = false;
    void fork() {
        if (!side || big_group < 0 || err != cudaSuccess) return;
        fail_here(cudaEventRecord(ev_fork, stream), "cudaEventRecord(fork)");
        fail_here(cudaStreamWaitEvent(side, ev_fork, 0), "cudaStreamWaitEvent(fork)");
        main_stream = stream;
        forked = err == cudaSuccess;
    }
    void select(int group) {  // the stream the launches of this group go to
        if (forked) stream = (group == big_group) ? main_stream : side;
    }
    void join() {
        if (!forked) return;
        stream = main_stream;
        forked = false;
        fail_here(cudaEventRecord(ev_join, side), "cudaEventRecord(join)");
        fail_here(cudaStreamWaitEvent(stream, ev_join, 0), "cudaStreamWaitEvent(join)");
    }
    void memset(void* p, int v, size_t bytes) {
        if (bytes == 0 || err != cudaSuccess) return;
        cudaError_t e = cudaMemsetAsync(p, v, bytes, stream);
        if (e != cudaSuccess && err == cudaSuccess) { err = e; err_where = "memset"; }
    }

    // ---- CUDA-graph capture of the step (small systems, flare_api.cu): `stream` is being captured.  A conditional
    // IF node lets the graph skip the whole candidate-list rebuild chain unless the device-side gate asks for it:
    //   h = cond_handle();  launch(kernel that calls cudaGraphSetConditional(h, need));  begin_if(h);
    //   ... launches of the body ...;  end_if();
    bool capturing = false;
    cudaStream_t body_stream = nullptr;  // side stream the IF body is captured on
    cudaStream_t outer_stream = nullptr;
    cudaGraphNode_t cond_node = nullptr;
    cudaGraphConditionalHandle cond_handle() {
        cudaGraphConditionalHandle h = 0;
        if (err != cudaSuccess) return h;
        cudaStreamCaptureStatus st;
        cudaGraph_t g = nullptr;
        const cudaGraphNode_t* deps = nullptr;
        size_t nd = 0;
        fail_here(cudaStreamGetCaptureInfo_v2(stream, &st, nullptr, &g, &deps, &nd), "cudaStreamGetCaptureInfo");
        if (err == cudaSuccess) fail_here(cudaGraphConditionalHandleCreate(&h, g, 0, cudaGraphCondAssignDefault), "cudaGraphConditionalHandleCreate");
        return h;
    }
    void begin_if(cudaGraphConditionalHandle h) {
        if (err != cudaSuccess) return;
        cudaStreamCaptureStatus st;
        cudaGraph_t g = nullptr;
        const cudaGraphNode_t* deps = nullptr;
        size_t nd = 0;
        fail_here(cudaStreamGetCaptureInfo_v2(stream, &st, nullptr, &g, &deps, &nd), "cudaStreamGetCaptureInfo");
        if (err != cudaSuccess) return;
        cudaGraphNodeParams p = {cudaGraphNodeTypeConditional};
        p.conditional.handle = h;
        p.conditional.type = cudaGraphCondTypeIf;
        p.conditional.size = 1;
        fail_here(cudaGraphAddNode(&cond_node, g, deps, nd, &p), "cudaGraphAddNode(conditional)");
        if (err != cudaSuccess) return;
        fail_here(cudaStreamBeginCaptureToGraph(body_stream, p.conditional.phGraph_out[0], nullptr, nullptr, 0,
                                                cudaStreamCaptureModeThreadLocal), "cudaStreamBeginCaptureToGraph");
        if (err != cudaSuccess) return;
        outer_stream = stream;
        stream = body_stream;
    }
    void end_if() {
        if (outer_stream == nullptr) return;
        cudaError_t e = cudaStreamEndCapture(body_stream, nullptr);
        stream = outer_stream;
        outer_stream = nullptr;
        fail_here(e, "cudaStreamEndCapture(conditional body)");
        if (err == cudaSuccess)
            fail_here(cudaStreamUpdateCaptureDependencies(stream, &cond_node, 1, cudaStreamSetCaptureDependencies),
                      "cudaStreamUpdateCaptureDependencies");
    }
};

// Device pointers carved out of the caller's workspace by flare_bind.
struct Workspace {
    // ---- persistent per-atom state (caller order) for flare_step
    double* x = nullptr;    // [N][3]
    double* v = nullptr;    // [N][3]
    double* f = nullptr;    // [N][3]
    double* e = nullptr;    // [N]
    double* var = nullptr;  // [N]
    int* types = nullptr;   // [N]
    // ---- neighbour stage
    int* flags = nullptr;         // [4] device error bits
    int* cell_cnt = nullptr;      // [n_cells_cap]
    int* cell_start = nullptr;    // [n_cells_cap+1]
    int* scan_tmp = nullptr;      // [n_cells_cap/1024+2]
    int* cell_of = nullptr;       // [N]
    int* rank_in_cell = nullptr;  // [N]
    int* order = nullptr;         // [N] sorted slot -> caller index
    AtomS* atoms = nullptr;       // [N] cell-sorted
    int* nbr_cnt = nullptr;       // [N]
    int* nbr_idx = nullptr;       // [N][mmax] sorted-space indices
    unsigned char* rev = nullptr;    // [N][mmax]
    unsigned char* nmask = nullptr;  // [N] neighbour-species bitmask
    int* group_hist = nullptr;    // [ceil(N/1024)][n_groups]
    int* group_start = nullptr;   // [n_groups+1]
    int* row_of = nullptr;        // [N] sorted atom -> quadratic-form row
    unsigned char* gid = nullptr; // [N] group id of each sorted atom
    int* atom_of_row = nullptr;   // [N]
    // ---- skin list (candidates within r_cut + skin, kept across evaluations; only with FLARE_OPT_SKIN > 0)
    int* skin_cnt = nullptr;               // [N]
    int* skin_idx = nullptr;               // [N][kSkinStride]
    unsigned char* skin_rev = nullptr;     // [N][kSkinStride] reverse index of the candidate list
    AtomS* ref = nullptr;                  // [N] sorted atoms at the time the list was built
    unsigned long long* hitmask = nullptr; // [N] bit s: candidate s passes the exact predicate
    int* skin_gate = nullptr;              // [1] non-zero: rebuild in this evaluation
    // ---- per-atom results in sorted order
    double* pairf = nullptr;  // [N][mmax][3]  dE_k/dr_kj
    double* e_s = nullptr;    // [N]
    double* v_s = nullptr;    // [N]
    // ---- chunk-sized intermediates (rows of the current chunk)
    double* A = nullptr;     // [chunk][NvL2]
    double* Bh = nullptr;    // [chunk][Pld]
    double* W = nullptr;     // [chunk][Pld]
    double* nrm = nullptr;   // [chunk] ||B||^2 of the unnormalised rows
    double* part = nullptr;  // [2][max_ntn][chunk]  partial row-dots of the energy / variance tiles
    // ---- reductions and scalars of the analysis / thermostat kernels
    double* red = nullptr;                 // [kRedBlocksMax][9] per-block partial sums
    double* scal = nullptr;                // [16]: [0..8] virial, [12..15] thermostat xi, eta, scale, K2
    unsigned long long* ascal = nullptr;   // [18] analysis outputs (max bits, count, coordination histogram)
    int* qf_counter = nullptr;             // [3 kMaxGroups] tile / block queues of the quadratic-form launches
    // ---- domain decomposition
    long long* tag = nullptr;  // [N] global atom id (travels with the atom)
    int* dom = nullptr;        // [kDomInts] counters, see kDom*
    int* send_idx = nullptr;   // [4][N/2 + 1024] send lists of the two exchange phases
    double* dom_ref = nullptr; // [N][3] positions at the last domain rebuild (caller order)
};
constexpr int kRedBlocksMax = 1184;

// One quadratic-form group: rows whose atoms share the matrix (and, in sparse mode, the component set).
struct GroupDesc {
    int P = 0;            // descriptor components of this group (all of them in dense mode)
    int K = 0;            // P padded to a multiple of 16 = reduction length and row length used
    int nb = 0;           // n8-blocks per tile (tile width 8*nb)
    int ntn = 0;          // tiles along N per matrix
    const double* beta = nullptr;   // device [ntn*8*nb][K] padded, symmetric
    const double* sigma = nullptr;  // same or nullptr
    const int* table = nullptr;     // device [P/(l_max+1)]: pair q -> nu1 | nu2<<8; component p = q*(l_max+1) + l
    const int* lut = nullptr;       // device [Nv*Nv]: (nu1,nu2) -> pair q (symmetric), -1 if not in the group
    unsigned mask = 0;              // neighbour species of the group (all species in dense mode)
    int nsp = 0;                    // popcount(mask)
    int Nc = 0;                     // nsp * n_max compact radial channels: compact index = rank(species) * n_max + n;
                                    // the group's components are the triangular enumeration over them (x l)
    unsigned sidx = 0;              // 4 bits per species: its rank within mask (15 = absent)
};

// Atoms per warp of the per-atom kernels: packing the neighbour lists of several atoms into 32-pair passes fills the
// lanes, but a small system is bound by the latency of one warp's chain, not by throughput: with fewer than ~2 warps
// per SM sub-partition at the full count, take fewer atoms per warp so that more warps (and SMs) share the rows.
inline int small_system_ta(int nrows, int warps_per_cta, int ta_max) {
    const int warps_wanted = 148 * 4 * 2;
    int ta = ta_max;
    while (ta > 1 && (nrows + ta - 1) / ta < warps_wanted) ta--;
    (void)warps_per_cta;
    return ta;
}

// What a per-(chunk, group) launch of the per-atom kernels needs (passed by value).
struct GroupRun {
    int g;          // group id: rows group_start[g] .. group_start[g+1], intersected with the chunk
    int row0, nrows;  // chunk = global rows [row0, row0 + nrows)
    int nsp, Nc;
    unsigned sidx;
    int P, K, ntn;
    const int* table;
};

inline GroupRun make_group_run(const GroupDesc& gd, int g, int row0, int nrows) {
    return GroupRun{g, row0, nrows, gd.nsp, gd.Nc, gd.sidx, gd.P, gd.K, gd.ntn, gd.table};
}

// What the per-atom kernels need to know about a group (device array indexed by group id).
struct GroupDev {
    int P;
    int K;
    int ntn;
    int pad_;
    const int* table;  // pair table, see GroupDesc
    const int* lut;    // pair lookup, see GroupDesc
};

// stage entry points (each enqueues kernels through the Launcher)
// skin > 0: keep a candidate list with cutoffs r_cut + skin across evaluations (list_valid: one exists for this
// order / box / types) and filter it with the exact predicate; skin = 0: rebuild everything every time.
void build_neighbors(Launcher& L, const Grid& g, const Basis& bs, const Workspace& ws, int n, const double* pos,
                     const int* types, int mmax, int sparse, int n_groups, double skin, bool list_valid,
                     double dom_trigger = 0.0,  // > 0: raise Workspace::dom[kDomNeed] once an atom has moved that far
                     double dom_limit = 0.0);   // > 0: raise kFlagHaloExceeded once an atom has moved that far

// Descriptor rows [row0,row0+nrows): compact A -> ws.A, UNNORMALISED B -> bh_out (row r at (r - row0)*ld),
// ||B||^2 -> nrm_out.  One launch per group.
void run_descriptors(Launcher& L, const Grid& g, const Basis& bs, const YNorm& yn, const Workspace& ws, int mmax,
                     const GroupDesc* groups, int n_groups, int row0, int nrows, double* bh_out, int ld,
                     double* nrm_out, bool write_A);

void run_qform(Launcher& L, const Workspace& ws, const GroupDesc* groups, int n_groups, int row0, int nrows, int ld,
               int chunk_cap, bool want_variance, int sm_count);

void run_backprop(Launcher& L, const Grid& g, const Basis& bs, const YNorm& yn, const Workspace& ws, int mmax,
                  const GroupDesc* groups, int n_groups, int row0, int nrows, int ld, int chunk_cap, int max_ntn,
                  bool want_variance);

void run_gather(Launcher& L, const Workspace& ws, int n, int mmax, double* e_out, double* f_out, double* var_out);

void run_kick_drift(Launcher& L, const Grid& g, int n, double* x, double* v, const double* f, const int* types,
                    const double* accel_half_dt /*[S] device: 0.5 dt kappa / m*/, double dt);
void run_kick(Launcher& L, int n, double* v, const double* f, const int* types, const double* accel_half_dt);

// analysis.cu: virial -> out9 (device), analysis -> out18 (device), one Nose-Hoover half step of length h
void run_virial(Launcher& L, const Grid& g, const Workspace& ws, int n, int mmax, double* out9);
void run_analyze(Launcher& L, const Grid& g, const Workspace& ws, int n, int mmax, bool have_var, double threshold,
                 int species_a, int species_b, double r_coord, bool want_coord, int* coord,
                 unsigned long long* out18);
void run_nh_half(Launcher& L, const Workspace& ws, int n, const double* mass_dev, double h, double gkT, double Q,
                 double* thermo);

// virial_static.cu: the virial with its partial sums in a static device array of the library (no workspace scratch,
// no allocation); at most kVirialStaticMaxAtoms atoms (= FLARE_VIRIAL_STATIC_MAX_ATOMS of the header)
constexpr int64_t kVirialStaticMaxAtoms = 4194304;
cudaError_t run_virial_static(Launcher& L, int device, const Grid& g, const Workspace& ws, int n, int mmax,
                              double* out9);

// domain.cu: selection / packing / compaction kernels of the domain decomposition (all sizes on the device)
void dom_select(Launcher& L, const Workspace& ws, const DomSel& s, int n_bound, int* list_lo, int* list_hi,
                int* list_stay, int cap);
void dom_commit_lists(Launcher& L, const Workspace& ws, int slot_lo, int slot_hi, int cap);
void dom_pack_full(Launcher& L, const Workspace& ws, const int* list, int cnt_slot, const double shift[3],
                   bool with_force, double* msg, int cap_rows);
void dom_append(Launcher& L, const Workspace& ws, const double* msg, int n_cap, int max_rows, int slot, bool owned);
void dom_compact_stay(Launcher& L, const Workspace& ws, const int* list_stay, int n_bound);
void dom_set_counts(Launcher& L, const Workspace& ws, int from_slot, bool to_local, bool to_owned);
void dom_pack_fwd(Launcher& L, const Workspace& ws, const int* list, int cnt, const double shift[3], double* msg);
void dom_unpack_fwd(Launcher& L, const Workspace& ws, const double* msg, int off, int cnt);

}  // namespace flare
