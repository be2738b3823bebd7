// qform.cu -- steps a4 + a5: the mapped mean E_i = d^T beta d and variance V_i = d^T Sigma d
// (Eq. 1-2), batched over the atoms of a group as a dense FP64 contraction
//     W[rows x K] = B^[rows x K] . M[K x K],   M = beta^(s) or Sigma^(s) (symmetric, K = padded P),
// on the FP64 tensor pipe (mma.sync.m8n8k4.f64 -> DMMA.8x8x4; tcgen05 has no f64 kind).
// The paper does this one atom per block as a mat-vec; here the descriptor rows of 64 atoms
// share every tile of the matrix.
//
// Tiling: CTA tile 64 rows x (8*NB) columns, 4 warps stacked along M (16 rows each), every warp spans
// the full tile width, so the row-dots of the epilogue never cross warps; two CTAs per SM, tiles taken
// from a device counter.  K is streamed in slabs of 16 through a 3-stage cp.async pipeline (the next
// tile's first slabs are requested before the epilogue); shared-memory rows are padded to 20 doubles so
// that the 8-byte fragment loads of a half-warp hit 16 distinct bank pairs.  Variance tiles use the
// symmetry of Sigma (upper 16 x 16 super-blocks only).
// Epilogue (fused): energy tiles store W = beta B (needed for dE/dB) and the partial row-dot
// sum_n W[r][n] B[r][n]; variance tiles store only the partial row-dot.  Partials of the ntn tiles
// of a row are summed in fixed order by the back-propagation kernel (deterministic, atomics-free).
// The rows hold the UNNORMALISED B; the 1/||B||^2 factor is applied by the back-propagation kernel.
#include <algorithm>
#include <type_traits>

#include "kernels.cuh"

namespace flare {

constexpr int kQfBK = 16;       // K slab
constexpr int kQfLds = 20;      // padded slab row (doubles)

struct QfArgs {
    const double* Bh;   // [chunk rows][ld]  (unnormalised B rows)
    double* W;          // [chunk rows][ld]
    double* part;       // [2][max_ntn][chunk_cap]
    const int* group_start;
    const double* beta;
    const double* sigma;  // may be null
    int g;                // group id
    int row0, nrows;      // chunk = global rows [row0, row0+nrows)
    int ld;
    int K;                // reduction length (multiple of 16)
    int ntn;              // tiles along N per matrix
    int n_mat;            // 1 (energy only) or 2 (+variance)
    int chunk_cap;
    int max_ntn;
    int* counter;         // tile queue of this launch (zeroed before it)
};

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src, int src_bytes) {
    unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s), "l"(gmem_src), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N)); }

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}

// WARPS warps stacked along M (16 rows each): CTA tile (16 WARPS) x (8 NB).  WARPS = 4 runs two CTAs per SM
// (3 stages each), so that one CTA's epilogue and pipeline refill overlap the other's DMMA main loop.
template <int WARPS> struct QfCfg {
    static constexpr int BM = 16 * WARPS;
    static constexpr int THREADS = 32 * WARPS;
    static_assert(WARPS == 4, "only the 4-warp tile is built (the 8-warp, one-CTA-per-SM variant of round 1 was slower)");
    static constexpr int STAGES = 3;
    static constexpr int MINB = 2;
};

template <int NB, int WARPS>
__global__ void __launch_bounds__(QfCfg<WARPS>::THREADS, QfCfg<WARPS>::MINB) k_qform(QfArgs a) {
    using C = QfCfg<WARPS>;
    constexpr int BN = 8 * NB;
    constexpr int BM = C::BM, THREADS = C::THREADS, STAGES = C::STAGES;
    extern __shared__ __align__(16) double smem[];
    double* As = smem;                               // [stages][BM][20]
    double* Bs = smem + STAGES * BM * kQfLds;        // [stages][BN][20]

    const int gs = max(a.group_start[a.g], a.row0);
    const int ge = min(a.group_start[a.g + 1], a.row0 + a.nrows);
    const int n_rows = ge - gs;
    if (n_rows <= 0) return;
    const int lrow0 = gs - a.row0;  // first local row of this group in the chunk buffers
    const int m_tiles = (n_rows + BM - 1) / BM;
    const int tiles_per_m = a.ntn * a.n_mat;
    const int total = m_tiles * tiles_per_m;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g8 = lane >> 2, t4 = lane & 3;
    const int nk = a.K / kQfBK;

    // tile -> (row block, matrix, column block), decoded ONCE per tile (the divisions are not paid per K slab)
    struct TileCtx {
        const double* Ag;  // first row of the tile in the B array
        const double* M;   // first row (n) of the tile's columns in the symmetric matrix
        int rows_here;
    };
    auto decode = [&](int tile) {
        const int mt = tile / tiles_per_m;
        const int rem = tile - mt * tiles_per_m;
        const int mat = rem / a.ntn;
        const int nt = rem - mat * a.ntn;
        TileCtx c;
        c.M = (mat == 0 ? a.beta : a.sigma) + (size_t)nt * BN * a.K;
        c.Ag = a.Bh + (size_t)(lrow0 + mt * BM) * a.ld;
        c.rows_here = min(BM, n_rows - mt * BM);
        return c;
    };
    // loads of one K slab of a tile into a stage
    auto load_stage = [&](const TileCtx& c, int kt, int stage) {
        const int k0 = kt * kQfBK;
        double* as = As + stage * BM * kQfLds;
        double* bs = Bs + stage * BN * kQfLds;
#pragma unroll
        for (int i = 0; i < (BM * 8) / THREADS; i++) {  // A slab: BM rows x 8 chunks of 16 B
            const int idx = tid + i * THREADS;
            const int r = idx >> 3, ch = idx & 7;
            const bool ok = r < c.rows_here;
            const double* src = c.Ag + (size_t)(ok ? r : 0) * a.ld + k0 + 2 * ch;
            cp_async16(as + r * kQfLds + 2 * ch, src, ok ? 16 : 0);
        }
        for (int idx = tid; idx < BN * 8; idx += THREADS) {  // B slab: BN rows x 8 chunks
            const int r = idx >> 3, ch = idx & 7;
            cp_async16(bs + r * kQfLds + 2 * ch, c.M + (size_t)r * a.K + k0 + 2 * ch, 16);
        }
    };
    // Variance tiles use the symmetry of Sigma: V = sum_{n,k} Sigma[n,k] d_n d_k only needs the 16 x 16 super-blocks with
    // n-block >= k-block, the strictly upper ones counted twice, so a variance tile stops at the K slab that holds its
    // last column and skips the column blocks left of the current slab (about half the DMMAs).  Energy tiles need all of
    // W = beta d (it feeds dE/dB), so they stay dense.
    auto tile_nk = [&](int tile) {
        const int rem = tile % tiles_per_m;
        const int mat = rem / a.ntn;
        const int nt = rem - mat * a.ntn;
        return mat == 0 ? nk : min(nk, (nt * BN + BN - 1) / kQfBK + 1);
    };
    auto prologue = [&](int tile) {
        const int nkt = tile_nk(tile);
        const TileCtx c = decode(tile);
#pragma unroll
        for (int s = 0; s < STAGES - 1; s++) {
            if (s < nkt) load_stage(c, s, s);
            cp_async_commit();
        }
    };

    // Tiles are handed out through a counter: variance tiles are cheaper than energy tiles, so a static assignment
    // (tile += gridDim.x keeps a CTA on one kind when the grid is even) left half of the CTAs idle at the end.
    __shared__ int s_tile;
    if (tid == 0) s_tile = atomicAdd(a.counter, 1);
    __syncthreads();
    int tile = s_tile;
    if (tile < total) prologue(tile);
    while (tile < total) {
        const int mt = tile / tiles_per_m;
        const int rem = tile - mt * tiles_per_m;
        const int mat = rem / a.ntn;
        const int nt = rem - mat * a.ntn;
        const int mrow0 = mt * BM;  // row offset inside the group

        double acc[2][NB][2];
#pragma unroll
        for (int h = 0; h < 2; h++)
#pragma unroll
            for (int nb = 0; nb < NB; nb++) { acc[h][nb][0] = 0.0; acc[h][nb][1] = 0.0; }

        const int nkt = tile_nk(tile);
        const int nB0 = (nt * BN) / kQfBK;  // first 16-wide super-block of the tile's columns
        const TileCtx ctx = decode(tile);
        for (int kt = 0; kt < nkt; kt++) {
            cp_async_wait<STAGES - 2>();
            __syncthreads();
            if (kt + STAGES - 1 < nkt) load_stage(ctx, kt + STAGES - 1, (kt + STAGES - 1) % STAGES);
            cp_async_commit();
            const double* as = As + (kt % STAGES) * BM * kQfLds + (warp * 16 + g8) * kQfLds + t4;
            const double* bs = Bs + (kt % STAGES) * BN * kQfLds + g8 * kQfLds + t4;
            if (mat == 0) {
#pragma unroll
                for (int ks = 0; ks < kQfBK / 4; ks++) {
                    const double a0 = as[4 * ks];
                    const double a1 = as[8 * kQfLds + 4 * ks];
#pragma unroll
                    for (int nb = 0; nb < NB; nb++) {
                        const double b = bs[nb * 8 * kQfLds + 4 * ks];
                        dmma884(acc[0][nb][0], acc[0][nb][1], a0, b);
                        dmma884(acc[1][nb][0], acc[1][nb][1], a1, b);
                    }
                }
            } else {
                // super-block of column block nb relative to the slab: rel = rel0 + nb / 2; < 0: not needed, 0: diagonal
                // (counted once), > 0: strictly upper (counted twice).  Skipping is decided per GROUP of 6 column blocks
                // (one warp-uniform branch, the 12 DMMAs inside stay one straight-line block); blocks of an active group
                // that are not needed run with a zero operand.
                const int rel0 = nB0 - kt;
#pragma unroll
                for (int ks = 0; ks < kQfBK / 4; ks++) {
                    const double a0 = as[4 * ks];
                    const double a1 = as[8 * kQfLds + 4 * ks];
                    const double a0d = 2.0 * a0, a1d = 2.0 * a1;
#pragma unroll
                    for (int gb = 0; gb < NB; gb += 6) {
                        constexpr int kLastOfGroup = 5;
                        if (rel0 + min(gb + kLastOfGroup, NB - 1) / 2 >= 0) {  // the group's last super-block is needed
#pragma unroll
                            for (int nb = gb; nb < gb + 6 && nb < NB; nb++) {
                                const int rel = rel0 + nb / 2;
                                const double x0 = rel < 0 ? 0.0 : (rel > 0 ? a0d : a0);
                                const double x1 = rel < 0 ? 0.0 : (rel > 0 ? a1d : a1);
                                const double b = bs[nb * 8 * kQfLds + 4 * ks];
                                dmma884(acc[0][nb][0], acc[0][nb][1], x0, b);
                                dmma884(acc[1][nb][0], acc[1][nb][1], x1, b);
                            }
                        }
                    }
                }
            }
        }
        // all warps are done with the stages: refill the pipeline for the next tile, so that its first
        // slabs arrive while this tile's epilogue runs
        __syncthreads();
        if (tid == 0) s_tile = atomicAdd(a.counter, 1);
        __syncthreads();
        const int next = s_tile;
        if (next < total) prologue(next);

        // ---- fused epilogue: W store (energy tiles) + partial row-dot with B of the same columns
        const int n0 = nt * BN;
        double* part = a.part + ((size_t)mat * a.max_ntn + nt) * a.chunk_cap;
#pragma unroll
        for (int h = 0; h < 2; h++) {
            const int r = mrow0 + warp * 16 + h * 8 + g8;  // row inside the group
            const bool rok = r < n_rows;
            const size_t lrow = (size_t)(lrow0 + r);
            double dot = 0.0;
            if (rok) {
                const double* __restrict__ brow = a.Bh + lrow * a.ld;
                double* __restrict__ wrow = a.W + lrow * a.ld;
                // the B loads of a batch are issued together (one L2 round trip per batch, not per column block)
                constexpr int CH = 6;
#pragma unroll
                for (int nb0 = 0; nb0 < NB; nb0 += CH) {
                    double2 bv[CH];
#pragma unroll
                    for (int c = 0; c < CH; c++) {
                        const int n = n0 + (nb0 + c) * 8 + 2 * t4;
                        bv[c] = (nb0 + c < NB && n < a.K) ? __ldg(reinterpret_cast<const double2*>(brow + n))
                                                          : make_double2(0.0, 0.0);
                    }
#pragma unroll
                    for (int c = 0; c < CH; c++) {
                        if (nb0 + c < NB) {
                            dot = fma(acc[h][nb0 + c][0], bv[c].x, dot);
                            dot = fma(acc[h][nb0 + c][1], bv[c].y, dot);
                        }
                    }
                }
                if (mat == 0) {
#pragma unroll
                    for (int nb = 0; nb < NB; nb++) {
                        const int n = n0 + nb * 8 + 2 * t4;
                        if (n < a.K)  // K is even, so n+1 < K too
                            *reinterpret_cast<double2*>(wrow + n) = make_double2(acc[h][nb][0], acc[h][nb][1]);
                    }
                }
            }
            dot += __shfl_xor_sync(kFull, dot, 1);
            dot += __shfl_xor_sync(kFull, dot, 2);
            if (rok && t4 == 0) part[lrow] = dot;
        }
        tile = next;
    }
    cp_async_wait<0>();
}

template <int NB, int WARPS>
static void launch_qform(Launcher& L, const QfArgs& a, int sm_count, long long max_m_rows) {
    using C = QfCfg<WARPS>;
    constexpr int BN = 8 * NB;
    const size_t smem = sizeof(double) * C::STAGES * (C::BM + BN) * kQfLds;
    L.ensure_smem(k_qform<NB, WARPS>, smem);
    // persistent grid: MINB CTAs per SM, but never more CTAs than the chunk could give tiles
    const long long max_tiles = ((max_m_rows + C::BM - 1) / C::BM) * a.ntn * a.n_mat;
    // resident CTAs per SM of this instantiation (narrow tiles need few registers: more than MINB fit)
    const int occ = L.occupancy(k_qform<NB, WARPS>, C::THREADS, smem, C::MINB);
    const long long cap = (long long)sm_count * occ;
    const int grid = (int)(max_tiles < cap ? max_tiles : cap);
    L.launch(k_qform<NB, WARPS>, dim3(grid), dim3(C::THREADS), smem, a);
}

// ------------------------------------------------------------------ K <= 144: matrix resident in shared memory
// For the small matrices (P = 144 after the species-sparse compaction: 98 % of the rows of the H2/Pt(111)
// workloads) the whole symmetric matrix fits in one SM's shared memory (144 x 148 doubles = 170 KB).  One persistent
// CTA per SM keeps ONE matrix (beta or Sigma) resident -- fetched once by per-row bulk copies (TMA, completion on an
// mbarrier) -- and its 16 warps work independently: a warp takes a block of 8 rows from a device queue, loads those
// rows of B straight into registers in A-fragment layout (8 x K doubles = 36 per lane at K = 144), and runs the
// whole K loop out of registers and the resident matrix, 48 output columns at a time (H = 2: 16-row blocks, 8 warps).  No operand ever waits on
// another warp: there is no barrier in the steady state, and a row's E (or V) is complete inside one warp, so no
// partial row-dots are left for later.  CTAs that run out of blocks of their matrix switch to the other one.
constexpr int kQrWarps = 8;  // warps per CTA at H = 2; 16 at H = 1
constexpr int kQrNB = 6;  // n8 blocks (48 columns) per pass: 24 accumulator doubles per lane

struct QrArgs {
    const double* Bh;
    double* W;
    double* part;  // [2][max_ntn][chunk_cap]; these groups have one tile along N
    const int* group_start;
    const double* beta;
    const double* sigma;  // may be null
    int g, row0, nrows, ld, n_mat, chunk_cap, max_ntn;
    int* counter;  // [2]: next 16-row block of the beta / Sigma queue (zeroed before the launch)
};

__device__ __forceinline__ void qr_mbar_init(uint64_t* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count));
}
__device__ __forceinline__ void qr_mbar_expect(uint64_t* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(bytes));
}
__device__ __forceinline__ void qr_bulk_row(void* smem_dst, const void* gmem_src, unsigned bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n" ::"r"(
                     (unsigned)__cvta_generic_to_shared(smem_dst)),
                 "l"(gmem_src), "r"(bytes), "r"((unsigned)__cvta_generic_to_shared(bar))
                 : "memory");
}
__device__ __forceinline__ void qr_mbar_wait(uint64_t* bar, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"((unsigned)__cvta_generic_to_shared(bar)),
        "r"(parity)
        : "memory");
}

template <int K16, int H>  // K = 16 K16; a warp's block is 8 H rows (H = 1: 16 warps per CTA, H = 2: 8 warps)
__global__ void __launch_bounds__(kQrWarps * 32 * (3 - H), 1) k_qform_res(QrArgs a) {
    constexpr int K = 16 * K16;
    constexpr int KS = K / 4;      // k4 steps
    constexpr int MS = K + 4;      // padded row of the resident matrix (= 4 mod 16: conflict-free operand loads)
    constexpr int NBT = K / 8;     // n8 blocks of the full width
    constexpr int NP = (NBT + kQrNB - 1) / kQrNB;  // passes over the columns
    constexpr int RB = 8 * H;      // rows per block
    extern __shared__ __align__(16) double smem[];
    double* Ms = smem;  // [K][MS]: row n holds M[n][0..K) = column n of the symmetric matrix
    __shared__ uint64_t bar;
    __shared__ int s_switch;

    const int gs = max(a.group_start[a.g], a.row0);
    const int ge = min(a.group_start[a.g + 1], a.row0 + a.nrows);
    const int n_rows = ge - gs;
    if (n_rows <= 0) return;
    const int lrow0 = gs - a.row0;
    const int n_items = (n_rows + RB - 1) / RB;
    const int tid = threadIdx.x, lane = tid & 31;
    const int g8 = lane >> 2, t4 = lane & 3;

    // which matrix this CTA starts with: Sigma items cost ~0.56 of a beta item (upper triangle only)
    int mat = (a.n_mat == 2 && ((blockIdx.x * 5) % 14) < 5) ? 1 : 0;
    unsigned phase = 0;
    if (tid == 0) {
        qr_mbar_init(&bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::);
    }
    __syncthreads();
    for (int round = 0; round < 2; round++) {
        // ---- fetch the matrix: K bulk copies of one row each into the padded rows
        // (one row per thread: issued by one thread alone the K copies take longer than a small system's whole K loop)
        if (tid < K) {
            asm volatile("fence.proxy.async.shared::cta;\n" ::);  // earlier generic-proxy reads of Ms are done (syncthreads)
            const double* M = mat == 0 ? a.beta : a.sigma;
            if (tid == 0) qr_mbar_expect(&bar, (unsigned)(K * K * sizeof(double)));
            qr_bulk_row(Ms + tid * MS, M + (size_t)tid * K, (unsigned)(K * sizeof(double)), &bar);
        }
        qr_mbar_wait(&bar, phase);
        phase ^= 1u;

        int* queue = a.counter + mat;
        double* part = a.part + (size_t)mat * a.max_ntn * a.chunk_cap;
        // the queue is read one block ahead: the atomic's round trip hides under the current block's K loop
        int next = 0;
        if (lane == 0) next = atomicAdd(queue, 1);
        for (;;) {
            const int item = __shfl_sync(kFull, next, 0);
            if (item >= n_items) break;
            if (lane == 0) next = atomicAdd(queue, 1);
            const int r_lo = item * RB + g8;  // rows of this lane inside the group: r_lo (and r_lo + 8)
            bool ok[H];
            const double* brow[H];
#pragma unroll
            for (int h = 0; h < H; h++) {
                ok[h] = r_lo + 8 * h < n_rows;
                brow[h] = a.Bh + (size_t)(lrow0 + (ok[h] ? r_lo + 8 * h : 0)) * a.ld;
            }
            // the rows of B in A-fragment layout: lane (g8, t4) holds B[row g8 (+8)][4 ks + t4]
            double af[H][KS];
#pragma unroll
            for (int ks = 0; ks < KS; ks++)
#pragma unroll
                for (int h = 0; h < H; h++) af[h][ks] = ok[h] ? __ldg(brow[h] + 4 * ks + t4) : 0.0;
            double dot[H];
#pragma unroll
            for (int h = 0; h < H; h++) dot[h] = 0.0;
            for (int p = 0; p < NP; p++) {
                double acc[H][kQrNB][2];
#pragma unroll
                for (int h = 0; h < H; h++)
#pragma unroll
                    for (int nb = 0; nb < kQrNB; nb++) { acc[h][nb][0] = 0.0; acc[h][nb][1] = 0.0; }
                const int nb0 = p * kQrNB;  // first n8 block of the pass
                const double* ms = Ms + (size_t)(nb0 * 8 + g8) * MS + t4;
                if (mat == 0) {
#pragma unroll
                    for (int ks = 0; ks < KS; ks++) {
#pragma unroll
                        for (int nb = 0; nb < kQrNB; nb++) {
                            if (NBT % kQrNB == 0 || nb0 + nb < NBT) {
                                const double b = ms[nb * 8 * MS + 4 * ks];
#pragma unroll
                                for (int h = 0; h < H; h++) dmma884(acc[h][nb][0], acc[h][nb][1], af[h][ks], b);
                            }
                        }
                    }
                } else {
                    // symmetric matrix: only the 16 x 16 super-blocks with column block >= k block, the strictly upper
                    // ones with a doubled operand.  One warp-uniform decision per k super-block picks a straight-line
                    // block of DMMAs (a per-DMMA condition ends up predicated, and a predicated-off DMMA still costs
                    // its pipe slot): `first` = first super-block of the pass that is needed, `diag` = it is the diagonal one.
                    const int sb0 = nb0 >> 1;  // first 16-column super-block of the pass
#pragma unroll
                    for (int sk = 0; sk < K16; sk++) {
                        auto blk = [&](auto first_c, auto diag_c) {
                            constexpr int FIRST = decltype(first_c)::value;
                            constexpr bool DIAG = decltype(diag_c)::value;
#pragma unroll
                            for (int k4 = 0; k4 < 4; k4++) {
                                const int ks = 4 * sk + k4;
#pragma unroll
                                for (int sb = FIRST; sb < kQrNB / 2; sb++) {
                                    if (NBT % kQrNB == 0 || nb0 + 2 * sb < NBT) {
#pragma unroll
                                        for (int e = 0; e < 2; e++) {
                                            const double b = ms[(2 * sb + e) * 8 * MS + 4 * ks];
#pragma unroll
                                            for (int h = 0; h < H; h++)
                                                dmma884(acc[h][2 * sb + e][0], acc[h][2 * sb + e][1],
                                                        (DIAG && sb == FIRST) ? af[h][ks] : 2.0 * af[h][ks], b);
                                        }
                                    }
                                }
                            }
                        };
                        using I0 = std::integral_constant<int, 0>;
                        using I1 = std::integral_constant<int, 1>;
                        using I2 = std::integral_constant<int, 2>;
                        const int d = sk - sb0;  // which super-block of the pass is the diagonal one
                        if (d < 0) blk(I0{}, std::false_type{});
                        else if (d == 0) blk(I0{}, std::true_type{});
                        else if (d == 1) blk(I1{}, std::true_type{});
                        else if (d == 2) blk(I2{}, std::true_type{});
                    }
                }
                // ---- epilogue of the pass: W store (beta) and the row-dot with B of the same columns.  B[row][c] of the
                // accumulator's columns c = 8 nb + 2 t4 + e sits in the A fragments of the same quad: lane t4' = c & 3 =
                // 2 (t4 & 1) + e, register ks = c >> 2 = 2 nb + (t4 >> 1) -- fetched by shuffles, not from memory
                const int src0 = (lane & ~3) | (2 * (t4 & 1));
                const bool hi = (t4 >> 1) != 0;
#pragma unroll
                for (int nb = 0; nb < kQrNB; nb++) {
                    if (NBT % kQrNB == 0 || nb0 + nb < NBT) {
                        const int c = (nb0 + nb) * 8 + 2 * t4;
#pragma unroll
                        for (int h = 0; h < H; h++) {
                            // the af index must be a compile-time constant and the pass index p is not: select over the passes
                            double lo_v = 0.0, hi_v = 0.0;
#pragma unroll
                            for (int pp = 0; pp < NP; pp++) {
                                if (pp == p) {
                                    const int kk = 2 * (pp * kQrNB + nb);
                                    if (kk + 1 < KS) { lo_v = af[h][kk]; hi_v = af[h][kk + 1]; }
                                }
                            }
                            const double x0 = __shfl_sync(kFull, lo_v, src0), y0 = __shfl_sync(kFull, hi_v, src0);
                            const double x1 = __shfl_sync(kFull, lo_v, src0 + 1), y1 = __shfl_sync(kFull, hi_v, src0 + 1);
                            dot[h] = fma(acc[h][nb][0], hi ? y0 : x0, dot[h]);
                            dot[h] = fma(acc[h][nb][1], hi ? y1 : x1, dot[h]);
                            if (mat == 0 && ok[h])
                                *reinterpret_cast<double2*>(a.W + (size_t)(lrow0 + r_lo + 8 * h) * a.ld + c) = make_double2(acc[h][nb][0], acc[h][nb][1]);
                        }
                    }
                }
            }
#pragma unroll
            for (int h = 0; h < H; h++) {
                dot[h] += __shfl_xor_sync(kFull, dot[h], 1);
                dot[h] += __shfl_xor_sync(kFull, dot[h], 2);
                if (t4 == 0 && ok[h]) part[lrow0 + r_lo + 8 * h] = dot[h];
            }
        }
        // ---- this matrix's queue is empty: help with the other one if it still has blocks
        if (a.n_mat < 2) break;
        __syncthreads();  // every warp is done with the resident matrix
        if (tid == 0) s_switch = (atomicAdd(a.counter + (mat ^ 1), 0) < n_items) ? 1 : 0;
        __syncthreads();
        if (!s_switch) break;
        mat ^= 1;
    }
}

// rows per warp block / 8.  The kernel is written for H = 1 or 2 (H = 2 halves the matrix reads from shared memory per
// row but needs 8 instead of 16 warps' worth of registers per warp); H = 1 was faster at every K <= 144 and is the only
// value instantiated -- the h-loops in the kernel unroll to one pass
constexpr int kQrH = 1;

template <int K16>
static void launch_qform_res(Launcher& L, const QrArgs& a, int sm_count) {
    constexpr int K = 16 * K16;
    constexpr int warps = kQrWarps * (3 - kQrH);
    const size_t smem = sizeof(double) * (size_t)K * (K + 4);
    L.ensure_smem(k_qform_res<K16, kQrH>, smem);
    // one CTA per SM; for small systems one CTA per block and matrix rather than 16 blocks per CTA: a block is ~5 us of
    // DMMA pipe time on one SM sub-partition, and a small step is bound by exactly such latencies
    const long long items = ((long long)a.nrows + 8 * kQrH - 1) / (8 * kQrH);
    (void)warps;
    const int grid = (int)std::max<long long>(1, std::min<long long>(sm_count, items * a.n_mat));
    L.launch(k_qform_res<K16, kQrH>, dim3(grid), dim3(warps * 32), smem, a);
}

void run_qform(Launcher& L, const Workspace& ws, const GroupDesc* groups, int n_groups, int row0, int nrows, int ld,
               int chunk_cap, bool want_variance, int sm_count) {
    if (nrows <= 0) return;
    int max_ntn = 0;
    for (int g = 0; g < n_groups; g++) max_ntn = groups[g].ntn > max_ntn ? groups[g].ntn : max_ntn;
    L.memset(ws.qf_counter, 0, sizeof(int) * 3 * kMaxGroups);  // tile queues; [kMaxGroups + 2 g]: the two block queues of k_qform_res
    for (int g = 0; g < n_groups; g++) {
        const GroupDesc& gd = groups[g];
        if (gd.K == 0 || gd.beta == nullptr) continue;
        QfArgs a;
        a.Bh = ws.Bh; a.W = ws.W; a.part = ws.part; a.group_start = ws.group_start;
        a.beta = gd.beta; a.sigma = gd.sigma;
        a.g = g; a.row0 = row0; a.nrows = nrows; a.ld = ld; a.K = gd.K; a.ntn = gd.ntn;
        a.n_mat = (want_variance && gd.sigma) ? 2 : 1;
        a.chunk_cap = chunk_cap; a.max_ntn = max_ntn;
        a.counter = ws.qf_counter + g;
        if (gd.K <= 144) {  // matrix resident in shared memory, warps independent
            QrArgs r;
            r.Bh = ws.Bh; r.W = ws.W; r.part = ws.part; r.group_start = ws.group_start;
            r.beta = gd.beta; r.sigma = gd.sigma;
            r.g = g; r.row0 = row0; r.nrows = nrows; r.ld = ld; r.n_mat = a.n_mat;
            r.chunk_cap = chunk_cap; r.max_ntn = max_ntn;
            r.counter = ws.qf_counter + kMaxGroups + 2 * g;
            switch (gd.K / 16) {
#define FLARE_CASE(KV)                            \
    case KV:                                      \
        launch_qform_res<KV>(L, r, sm_count);     \
        break;
                FLARE_CASE(1) FLARE_CASE(2) FLARE_CASE(3) FLARE_CASE(4) FLARE_CASE(5) FLARE_CASE(6) FLARE_CASE(7)
                FLARE_CASE(8) FLARE_CASE(9)
#undef FLARE_CASE
                default: break;
            }
            continue;
        }
        switch (gd.nb) {
#define FLARE_CASE(NBV)                                                   \
    case NBV:                                                             \
        launch_qform<NBV, 4>(L, a, sm_count, nrows);                      \
        break;
            // even widths only (choose_tiles): a tile starts on a 16-column super-block
            FLARE_CASE(2) FLARE_CASE(4) FLARE_CASE(6) FLARE_CASE(8) FLARE_CASE(10)
            FLARE_CASE(12) FLARE_CASE(14) FLARE_CASE(16) FLARE_CASE(18)
#undef FLARE_CASE
            default: if (L.err == cudaSuccess) { L.err = cudaErrorInvalidValue; L.err_where = "qform tile width"; } break;
        }
    }
}

}  // namespace flare
