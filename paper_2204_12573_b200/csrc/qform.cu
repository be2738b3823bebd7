// qform.cu -- steps a4 + a5: the mapped mean E_i = d^T beta d and variance V_i = d^T Sigma d
// (Eq. 1-2), batched over the atoms of a group as a dense FP64 contraction
//     W[rows x K] = B^[rows x K] . M[K x K],   M = beta^(s) or Sigma^(s) (symmetric, K = padded P),
// on the FP64 tensor pipe (mma.sync.m8n8k4.f64 -> DMMA.8x8x4; tcgen05 has no f64 kind).
// The paper does this one atom per block as a mat-vec; here the descriptor rows of up to
// 128 atoms share every tile of the matrix.
//
// Tiling: CTA tile 128 rows x (8*NB) columns, 8 warps stacked along M (16 rows each), every warp
// spans the full tile width, so the row-dots of the epilogue never cross warps.  K is streamed in
// slabs of 16 through a 4-stage cp.async pipeline; shared-memory rows are padded to 20 doubles so
// that the 8-byte fragment loads of a half-warp hit 16 distinct banks pairs.
// Epilogue (fused): energy tiles store W (needed for dE/dB) and the partial row-dot
// sum_n W[r][n] B^[r][n]; variance tiles store only the partial row-dot.  Partials of the ntn tiles
// of a row are summed in fixed order by the back-propagation kernel (deterministic, atomics-free).
#include "kernels.cuh"

namespace flare {

constexpr int kQfBM = 128;      // rows per CTA tile
constexpr int kQfBK = 16;       // K slab
constexpr int kQfLds = 20;      // padded slab row (doubles)
constexpr int kQfStages = 4;
constexpr int kQfThreads = 256;

struct QfArgs {
    const double* Bh;   // [chunk rows][ld]
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

template <int NB>
__global__ void __launch_bounds__(kQfThreads, 1) k_qform(QfArgs a) {
    constexpr int BN = 8 * NB;
    extern __shared__ __align__(16) double smem[];
    double* As = smem;                                     // [stages][128][20]
    double* Bs = smem + kQfStages * kQfBM * kQfLds;        // [stages][BN][20]

    const int gs = max(a.group_start[a.g], a.row0);
    const int ge = min(a.group_start[a.g + 1], a.row0 + a.nrows);
    const int n_rows = ge - gs;
    if (n_rows <= 0) return;
    const int lrow0 = gs - a.row0;  // first local row of this group in the chunk buffers
    const int m_tiles = (n_rows + kQfBM - 1) / kQfBM;
    const int tiles_per_m = a.ntn * a.n_mat;
    const int total = m_tiles * tiles_per_m;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g8 = lane >> 2, t4 = lane & 3;
    const int nk = a.K / kQfBK;

    for (int tile = blockIdx.x; tile < total; tile += gridDim.x) {
        const int mt = tile / tiles_per_m;
        const int rem = tile - mt * tiles_per_m;
        const int mat = rem / a.ntn;
        const int nt = rem - mat * a.ntn;
        const double* M = (mat == 0 ? a.beta : a.sigma) + (size_t)nt * BN * a.K;  // rows n of the symmetric matrix
        const int mrow0 = mt * kQfBM;  // row offset inside the group
        const double* Ag = a.Bh + (size_t)(lrow0 + mrow0) * a.ld;
        const int rows_here = min(kQfBM, n_rows - mrow0);

        double acc[2][NB][2];
#pragma unroll
        for (int h = 0; h < 2; h++)
#pragma unroll
            for (int nb = 0; nb < NB; nb++) { acc[h][nb][0] = 0.0; acc[h][nb][1] = 0.0; }

        auto load_stage = [&](int kt, int stage) {
            const int k0 = kt * kQfBK;
            double* as = As + stage * kQfBM * kQfLds;
            double* bs = Bs + stage * BN * kQfLds;
            // A slab: 128 rows x 8 chunks of 16 B
#pragma unroll
            for (int i = 0; i < (kQfBM * 8) / kQfThreads; i++) {
                const int idx = tid + i * kQfThreads;
                const int r = idx >> 3, c = idx & 7;
                const bool ok = r < rows_here;
                const double* src = Ag + (size_t)(ok ? r : 0) * a.ld + k0 + 2 * c;
                cp_async16(as + r * kQfLds + 2 * c, src, ok ? 16 : 0);
            }
            // B slab: BN rows x 8 chunks
            for (int idx = tid; idx < BN * 8; idx += kQfThreads) {
                const int r = idx >> 3, c = idx & 7;
                cp_async16(bs + r * kQfLds + 2 * c, M + (size_t)r * a.K + k0 + 2 * c, 16);
            }
        };

        __syncthreads();  // previous tile's smem reads are done
#pragma unroll
        for (int s = 0; s < kQfStages - 1; s++) {
            if (s < nk) load_stage(s, s);
            cp_async_commit();
        }
        for (int kt = 0; kt < nk; kt++) {
            cp_async_wait<kQfStages - 2>();
            __syncthreads();
            if (kt + kQfStages - 1 < nk) load_stage(kt + kQfStages - 1, (kt + kQfStages - 1) % kQfStages);
            cp_async_commit();
            const double* as = As + (kt % kQfStages) * kQfBM * kQfLds + (warp * 16 + g8) * kQfLds + t4;
            const double* bs = Bs + (kt % kQfStages) * BN * kQfLds + g8 * kQfLds + t4;
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
        }
        cp_async_wait<0>();

        // ---- fused epilogue: W store (energy tiles) + partial row-dot with B^ of the same columns
        const int n0 = nt * BN;
        double* part = a.part + ((size_t)mat * a.max_ntn + nt) * a.chunk_cap;
#pragma unroll
        for (int h = 0; h < 2; h++) {
            const int r = mrow0 + warp * 16 + h * 8 + g8;  // row inside the group
            const bool rok = r < n_rows;
            const size_t lrow = (size_t)(lrow0 + r);
            double dot = 0.0;
            if (rok) {
                const double* brow = a.Bh + lrow * a.ld;
                double* wrow = a.W + lrow * a.ld;
#pragma unroll
                for (int nb = 0; nb < NB; nb++) {
                    const int n = n0 + nb * 8 + 2 * t4;
                    if (n < a.K) {  // K is even, so n+1 < K too
                        const double2 bv = *reinterpret_cast<const double2*>(brow + n);
                        dot = fma(acc[h][nb][0], bv.x, dot);
                        dot = fma(acc[h][nb][1], bv.y, dot);
                        if (mat == 0) *reinterpret_cast<double2*>(wrow + n) = make_double2(acc[h][nb][0], acc[h][nb][1]);
                    }
                }
            }
            dot += __shfl_xor_sync(kFull, dot, 1);
            dot += __shfl_xor_sync(kFull, dot, 2);
            if (rok && t4 == 0) part[lrow] = dot;
        }
    }
}

template <int NB>
static void launch_qform(Launcher& L, const QfArgs& a, int grid) {
    constexpr int BN = 8 * NB;
    const size_t smem = sizeof(double) * kQfStages * (kQfBM + BN) * kQfLds;
    static bool configured = false;
    if (!configured) {
        cudaFuncSetAttribute(k_qform<NB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        configured = true;
    }
    L.launch(k_qform<NB>, dim3(grid), dim3(kQfThreads), smem, a);
}

void run_qform(Launcher& L, const Workspace& ws, const GroupDesc* groups, int n_groups, int row0, int nrows, int ld,
               int chunk_cap, bool want_variance, int sm_count) {
    if (nrows <= 0) return;
    int max_ntn = 0;
    for (int g = 0; g < n_groups; g++) max_ntn = groups[g].ntn > max_ntn ? groups[g].ntn : max_ntn;
    for (int g = 0; g < n_groups; g++) {
        const GroupDesc& gd = groups[g];
        if (gd.K == 0 || gd.beta == nullptr) continue;
        QfArgs a;
        a.Bh = ws.Bh; a.W = ws.W; a.part = ws.part; a.group_start = ws.group_start;
        a.beta = gd.beta; a.sigma = gd.sigma;
        a.g = g; a.row0 = row0; a.nrows = nrows; a.ld = ld; a.K = gd.K; a.ntn = gd.ntn;
        a.n_mat = (want_variance && gd.sigma) ? 2 : 1;
        a.chunk_cap = chunk_cap; a.max_ntn = max_ntn;
        // persistent grid: one CTA per SM, but never more CTAs than the chunk could give tiles
        long long max_tiles = (long long)((nrows + kQfBM - 1) / kQfBM) * gd.ntn * a.n_mat;
        int grid = (int)(max_tiles < sm_count ? max_tiles : sm_count);
        switch (gd.nb) {
#define FLARE_CASE(NBV) case NBV: launch_qform<NBV>(L, a, grid); break;
            FLARE_CASE(2) FLARE_CASE(4) FLARE_CASE(6) FLARE_CASE(8) FLARE_CASE(9) FLARE_CASE(10) FLARE_CASE(11)
            FLARE_CASE(12) FLARE_CASE(13) FLARE_CASE(14) FLARE_CASE(15) FLARE_CASE(16) FLARE_CASE(17) FLARE_CASE(18)
#undef FLARE_CASE
            default: if (L.err == cudaSuccess) { L.err = cudaErrorInvalidValue; L.err_where = "qform tile width"; } break;
        }
    }
}

// ------------------------------------------------------------------ FP64 DMMA issue peak (roofline denominator)
__global__ void k_dmma_peak(double* out, int iters, double a, double b) {
    double c[8][2];
#pragma unroll
    for (int i = 0; i < 8; i++) { c[i][0] = threadIdx.x; c[i][1] = i; }
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int i = 0; i < 8; i++) dmma884(c[i][0], c[i][1], a, b);
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 8; i++) s += c[i][0] + c[i][1];
    if (s == 123.456) out[0] = s;
}

double measure_dmma_peak(int device) {
    if (cudaSetDevice(device) != cudaSuccess) return -1.0;
    cudaDeviceProp p;
    if (cudaGetDeviceProperties(&p, device) != cudaSuccess) return -1.0;
    double* out = nullptr;
    if (cudaMalloc(&out, 8) != cudaSuccess) return -1.0;
    const int blocks = p.multiProcessorCount * 2, threads = 256, iters = 1 << 14;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    k_dmma_peak<<<blocks, threads>>>(out, iters, 1.0000001, 1e-9);
    cudaDeviceSynchronize();
    float best = 1e30f;
    for (int r = 0; r < 5; r++) {
        cudaEventRecord(e0);
        k_dmma_peak<<<blocks, threads>>>(out, iters, 1.0000001, 1e-9);
        cudaEventRecord(e1);
        cudaEventSynchronize(e1);
        float ms;
        cudaEventElapsedTime(&ms, e0, e1);
        if (ms < best) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(out);
    if (cudaGetLastError() != cudaSuccess) return -1.0;
    const double flops = 2.0 * 256 * 8 * (double)iters * blocks * (threads / 32);
    return flops / (best * 1e-3) * 1e-12;
}

}  // namespace flare
