// virial_static.cu -- flare_virial_static (include/flare_b200.h): the virial reduction of analysis.cu for hosts
// that must not allocate device memory and cannot spare workspace either.
//
// Who that is.  This library is meant to sit inside somebody else's MD program.  Such a program usually grabs its
// device memory once, up front, through its own pool (on the 10 M-atom configuration nearly all of the 180 GB), and
// from then on a cudaMalloc from inside a plug-in is a bug: it can fail because nothing is left, it stalls every
// stream of the device while the driver maps the memory (cudaFree likewise), and some hosts simply forbid it -- a
// pressure coupling that runs every step, a monitoring hook with a latency budget, a process that locked its
// memory limits after start-up.  Every other call of this library meets that by borrowing scratch from the
// workspace the caller bound; this one needs nothing from the caller but the 9 doubles of the result: its partial
// sums live in a fixed array inside the library image.
//
// What it costs.  kStaticRows x 9 doubles = 147 456 bytes of device memory on every GPU on which the library's
// module gets loaded, from that moment until the process exits, whether or not the call is ever made; and a ceiling
// of kStaticMaxAtoms atoms per call (one row per tile of kStaticTile atoms).
//
// Sharing.  There is ONE array per device and every call on that device uses it, whatever the context or stream.
// Calls that can overlap on the GPU (two streams, two host threads with their own contexts) overwrite each other's
// partial sums: the caller orders them (same stream, or an event).  Nothing in the array has to start at zero:
// stage 1 writes rows [0, n_rows) in full before stage 2, enqueued behind it on the same stream, reads exactly
// those rows, so whatever an earlier (larger) call left in the rows above is never looked at.
//
// The summation order is fixed (atom -> warp -> tile -> result), so repeated calls give bit-identical results; it
// is a different order from flare_get_virial's grid-stride assignment, so the two agree to rounding, not bit by bit.
#include <mutex>

#include "kernels.cuh"

namespace flare {

constexpr int kStaticTile = 2048;  // atoms per stage-1 block (8 warps x 256 atoms)
constexpr int kStaticRows = 2048;  // rows of 9 partial sums the array holds
constexpr int kStaticThreads = 256;
static_assert((int64_t)kStaticTile * kStaticRows == kVirialStaticMaxAtoms, "header constant out of step");

// In HOST code this name is only a handle for cudaGetSymbolAddress / cudaMemcpyToSymbol; it is not a device
// address and must never be handed to a kernel as a pointer.  Device code may use it directly.
static __device__ __align__(256) double g_virial_rows[kStaticRows * 9];

namespace {

// fixed-order block sum of 9 values; result valid in thread 0
__device__ __forceinline__ void tile_sum9(double (&v)[9], double* sm /*[8][9]*/) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
    for (int q = 0; q < 9; q++) v[q] = warp_sum(v[q]);
    if (lane == 0)
#pragma unroll
        for (int q = 0; q < 9; q++) sm[w * 9 + q] = v[q];
    __syncthreads();
    if (threadIdx.x == 0)
#pragma unroll
        for (int q = 0; q < 9; q++) {
            double t = 0.0;
            for (int ww = 0; ww < kStaticThreads / 32; ww++) t += sm[ww * 9 + q];
            v[q] = t;
        }
}

// stage 1: block b sums sum_j f_kj (x) r_kj over the atoms k of tile b and writes row b (always, also when the
// tile's atoms have no neighbours: stage 2 relies on every row below n_rows being freshly written)
__global__ void __launch_bounds__(kStaticThreads)
k_virial_tile(Grid g, int n, int mmax, const AtomS* __restrict__ atoms, const int* __restrict__ nbr_cnt,
              const int* __restrict__ nbr_idx, const double* __restrict__ pairf, double* __restrict__ rows) {
    __shared__ double sm[(kStaticThreads / 32) * 9];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    double v[9];
#pragma unroll
    for (int q = 0; q < 9; q++) v[q] = 0.0;
    const int k0 = blockIdx.x * kStaticTile;
    const int k1 = min(n, k0 + kStaticTile);
    for (int k = k0 + w; k < k1; k += kStaticThreads / 32) {
        const AtomS me = load_atom(atoms + k);
        const int cnt = nbr_cnt[k];
        for (int s = lane; s < cnt; s += 32) {
            const AtomS o = load_atom(atoms + nbr_idx[(size_t)k * mmax + s]);
            double d[3];
            displacement(g, me, o, d[0], d[1], d[2]);
            const double* pf = pairf + ((size_t)k * mmax + s) * 3;
#pragma unroll
            for (int a = 0; a < 3; a++)
#pragma unroll
                for (int b = 0; b < 3; b++) v[3 * a + b] = fma(pf[a], d[b], v[3 * a + b]);
        }
    }
    tile_sum9(v, sm);
    if (threadIdx.x == 0)
#pragma unroll
        for (int q = 0; q < 9; q++) rows[(size_t)blockIdx.x * 9 + q] = v[q];
}

// stage 2: one block adds rows [0, n_rows) in a fixed order -> out[9]
__global__ void __launch_bounds__(kStaticThreads)
k_virial_rows_sum(int n_rows, const double* __restrict__ rows, double* __restrict__ out) {
    __shared__ double sm[(kStaticThreads / 32) * 9];
    double v[9];
#pragma unroll
    for (int q = 0; q < 9; q++) v[q] = 0.0;
    for (int b = threadIdx.x; b < n_rows; b += kStaticThreads)
#pragma unroll
        for (int q = 0; q < 9; q++) v[q] += rows[(size_t)b * 9 + q];
    tile_sum9(v, sm);
    if (threadIdx.x == 0)
#pragma unroll
        for (int q = 0; q < 9; q++) out[q] = v[q];
}

// Device address of g_virial_rows, looked up once per device.  cudaGetSymbolAddress answers for the CURRENT device
// (each device that loads the module has its own copy of the array), so the table is indexed by ordinal and filled
// with that device current.  The lookup allocates nothing, but the first one on a device may make the runtime load
// the module there -- which is why the first call belongs before any stream capture.
constexpr int kMaxDeviceTable = 64;
std::mutex g_addr_mutex;
double* g_rows_addr[kMaxDeviceTable] = {};

cudaError_t static_rows_address(int device, double** out) {
    int cur = -1;
    cudaError_t e = cudaGetDevice(&cur);
    if (e != cudaSuccess) return e;
    if (cur != device) {
        e = cudaSetDevice(device);
        if (e != cudaSuccess) return e;
    }
    const bool cached = device >= 0 && device < kMaxDeviceTable;
    if (cached) {
        std::lock_guard<std::mutex> lock(g_addr_mutex);
        if (g_rows_addr[device]) { *out = g_rows_addr[device]; return cudaSuccess; }
    }
    double* p = nullptr;
    e = cudaGetSymbolAddress((void**)&p, g_virial_rows);
    if (e != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    if (cached) {
        std::lock_guard<std::mutex> lock(g_addr_mutex);
        g_rows_addr[device] = p;
    }
    *out = p;
    return cudaSuccess;
}

}  // namespace

// Enqueue the two stages on L's stream.  n in [0, kVirialStaticMaxAtoms] (checked by the caller, re-checked here);
// out9 is a DEVICE pointer.  Calls no allocating routine: one symbol lookup (first call per device), then launches.
cudaError_t run_virial_static(Launcher& L, int device, const Grid& g, const Workspace& ws, int n, int mmax,
                              double* out9) {
    if (n < 0 || (int64_t)n > kVirialStaticMaxAtoms) return cudaErrorInvalidValue;
    if (n == 0) return cudaMemsetAsync(out9, 0, sizeof(double) * 9, L.stream);
    double* rows = nullptr;
    cudaError_t e = static_rows_address(device, &rows);
    if (e != cudaSuccess) return e;
    const int n_rows = (n + kStaticTile - 1) / kStaticTile;
    L.launch(k_virial_tile, dim3(n_rows), dim3(kStaticThreads), 0, g, n, mmax, (const AtomS*)ws.atoms,
             (const int*)ws.nbr_cnt, (const int*)ws.nbr_idx, (const double*)ws.pairf, rows);
    L.launch(k_virial_rows_sum, dim3(1), dim3(kStaticThreads), 0, n_rows, (const double*)rows, out9);
    return L.err;
}

}  // namespace flare
