// common.cuh -- shared device-side types and helpers of the FLARE B200 kernels.
// (Shares nothing with oracle/: every formula here is restated from DESIGN.md section 2.)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace flare {

constexpr int kMaxSpecies = 8;
constexpr int kMaxNmax = 16;
constexpr int kMaxLmax = 6;
constexpr int kWarp = 32;
constexpr unsigned kFull = 0xffffffffu;

// Error bits raised by kernels into FlareCtx::d_flags[0]
constexpr int kFlagNeighborOverflow = 1;
constexpr int kFlagNonFinite = 2;        // a position is NaN/Inf
constexpr int kFlagBadType = 4;          // a species index outside 0..S-1 (stored as 0 so that indexing stays in bounds)
constexpr int kFlagNonFiniteResult = 8;  // an energy, force or variance came out NaN/Inf
constexpr int kFlagDomainOverflow = 16;  // domain decomposition: a message, a send list or the bound capacity is too small
constexpr int kFlagHaloExceeded = 32;    // domain decomposition: an atom has moved further since the last rebuild than the ghost shell covers

// One atom in cell-sorted order: wrapped position, species, index in the caller's order.
struct __align__(32) AtomS {
    double x, y, z;
    int type;
    int orig;
};
static_assert(sizeof(AtomS) == 32, "AtomS must be one 32-byte sector");

// Orthorhombic box + cell grid (R6, R7).  Passed by value to kernels.
struct Grid {
    double L[3];       // box lengths
    double half[3];    // 0.5*L
    double inv_cw[3];  // 1 / cell width
    int pbc[3];
    int nc[3];      // cells per dimension
    int stride[3];  // linear cell index = sum c[d]*stride[d]; the dimension with stride 1 is "fast"
    int fast;       // dimension with stride 1
    int slow0, slow1;
    int n_cells;
};

// Model constants needed by the per-pair basis (passed by value).
struct Basis {
    int S, n_max, l_max;
    int L2;      // (l_max+1)^2
    int Nv;      // S*n_max
    int NvL2;    // Nv*L2
    int P;       // descriptors
    int Pld;     // padded row length of B^/W rows (multiple of 16)
    double rc[kMaxSpecies * kMaxSpecies];
    double rc2[kMaxSpecies * kMaxSpecies];
    double irc[kMaxSpecies * kMaxSpecies];  // 1 / r_cut
};

// ------------------------------------------------------------------ canonical geometry (R6)
// Every operation individually rounded (no FMA contraction) so that neighbour sets are
// bit-identical to any other implementation of the same canonical formulas.

__device__ __forceinline__ double wrap_coord(double x, double L) {
    double q = floor(__ddiv_rn(x, L));
    double w = __dsub_rn(x, __dmul_rn(L, q));
    if (w >= L) w = 0.0;
    if (w < 0.0) w = 0.0;
    return w;
}

__device__ __forceinline__ double min_image(double d, double L, double half, int pbc) {
    // selects, not branches (same values: each candidate is one rounded operation on d)
    const double lo = __dsub_rn(d, L), hi = __dadd_rn(d, L);
    const double w = d > half ? lo : (d < -half ? hi : d);
    return pbc ? w : d;
}

__device__ __forceinline__ double dist2_canonical(double dx, double dy, double dz) {
    return __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
}

__device__ __forceinline__ void displacement(const Grid& g, const AtomS& a, const AtomS& b, double& dx, double& dy,
                                             double& dz) {
    dx = min_image(__dsub_rn(b.x, a.x), g.L[0], g.half[0], g.pbc[0]);
    dy = min_image(__dsub_rn(b.y, a.y), g.L[1], g.half[1], g.pbc[1]);
    dz = min_image(__dsub_rn(b.z, a.z), g.L[2], g.half[2], g.pbc[2]);
}

__device__ __forceinline__ AtomS load_atom(const AtomS* p) {
    // two 16-byte loads of one 32-byte sector
    const double2* q = reinterpret_cast<const double2*>(p);
    double2 a = __ldg(q);
    double2 b = __ldg(q + 1);
    AtomS r;
    r.x = a.x; r.y = a.y; r.z = b.x;
    long long bits = __double_as_longlong(b.y);
    r.type = (int)(bits & 0xffffffffll);
    r.orig = (int)(bits >> 32);
    return r;
}

// ------------------------------------------------------------------ warp reductions
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(kFull, v, o);
    return v;
}

}  // namespace flare
