// common.cuh -- lattice parameters, Philox4x32-10 and small device helpers shared by the sm_100a kernels.
// Part of libswb200 (include/swb200.h).  Shares nothing with oracle/.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace swb {

// Strip of the one-level decomposition ("tiles of B_x x B_y spins", P:84 B_x >> B_y for coalescing).
// k_scan: one WARP labels a TW x TH strip, lane -> 4 consecutive columns (one 32-bit word of int8 spins, one 128-bit
// vector of int32 labels), rows in sequence.  k_final: one CTA of FIN_THREADS threads per strip.
#ifndef SWB_TH_LOG
#define SWB_TH_LOG 5
#endif
constexpr int TW_LOG = 7, TH_LOG = SWB_TH_LOG;           // (TH = 16 needs SWB_FIN_THREADS = 128: k_final's warps own 4 rows each)
constexpr int TW = 1 << TW_LOG;
constexpr int TH = 1 << TH_LOG;
#ifndef SWB_SCAN_WARPS
#define SWB_SCAN_WARPS 4
#endif
#ifndef SWB_FIN_THREADS
#define SWB_FIN_THREADS 256
#endif
constexpr int SCAN_WARPS = SWB_SCAN_WARPS;               // strips per k_scan CTA (horizontally adjacent)
constexpr int SCAN_THREADS = 32 * SCAN_WARPS;
constexpr int FIN_THREADS = SWB_FIN_THREADS;
constexpr int FIN_WARPS = FIN_THREADS / 32;
#ifndef SWB_FIN_MIN_CTAS
#define SWB_FIN_MIN_CTAS (2048 / SWB_FIN_THREADS)
#endif
constexpr int FIN_MIN_CTAS = SWB_FIN_MIN_CTAS;
#ifndef SWB_FIN_MLP
#define SWB_FIN_MLP 2
#endif
constexpr int FIN_MLP = SWB_FIN_MLP;                     // strip-local roots a k_final lane resolves at a time
#ifndef SWB_GEN_ROWS
#define SWB_GEN_ROWS 0
#endif
constexpr int GEN_ROWS = SWB_GEN_ROWS;                   // rows of every 4 whose bond draws k_final computes one sweep ahead           // resident k_final CTAs per SM the register budget is set for
static_assert(TW == 128, "lane -> 4 columns, 32 lanes");
static_assert(TW * TH <= 65536, "strip-local indices are kept in uint16");
static_assert(TH % FIN_WARPS == 0 && 4 * (TH / FIN_WARPS) <= 32, "k_final keeps one bit per site of a thread in a 32-bit mask");

enum : uint32_t { DOM_INIT = 0, DOM_BOND = 1, DOM_FLIP = 2, DOM_WSEED = 3 };

// Everything a kernel needs to know about the lattice and the random stream; passed by value (constant bank).
struct Params {
    int32_t  L;          // edge length, multiple of 4
    int32_t  N;          // L*L <= 2^30
    int32_t  logL;       // log2(L) if L is a power of two, else -1
    int32_t  sbit;       // k_final keeps a cluster's new state above this bit of its label: 28 if N <= 2^28, else 30
    int32_t  q;          // number of Potts states (2 = Ising storage +-1)
    int32_t  ntx, nty;   // number of tile columns / rows
    uint32_t T;          // bond threshold floor(p 2^32)
    uint32_t t_lo, t_hi; // step counter
    uint32_t u_lo, u_hi; // step counter + 1 (k_final computes the bond draws of the next sweep)
    uint32_t k0[10];     // Philox round keys: k0[r] = seed_lo + r * 0x9E3779B9
    uint32_t k1[10];     //                    k1[r] = seed_hi + r * 0xBB67AE85
    uint32_t negT;       // 2^32 - T (mod 2^32): u + negT carries iff u >= T, for T != 0 (scan_kernel.cuh shift_in_ge)
    uint32_t dmask;      // 0xFF; 0 if T = 0 (no bond is ever active)
    int32_t  H;          // rows of the label array seen as H rows of L sites: L (square lattice) or L*L (simple cubic)
    int32_t  n3x, n3y, n3z;   // simple cubic lattice: number of tiles per direction (cubic_kernels.cuh), else 0
    int32_t  ty0, nband;      // row band of a multi-GPU run (band_kernels.cuh): first strip row and number of strip rows this
                              // handle works on; 0 and nty for the whole lattice
    uint32_t T_flip;          // few-cluster step (k_final<MODE_FEW>): a selected cluster is flipped iff its draw is < T_flip
    int32_t  few_mask;        // ... and the table of selected roots has few_mask + 1 slots (a power of two)
};

// Philox4x32-10 (Salmon et al., SC'11).  c1,c2,c3 are warp-uniform in every use here (step counter and domain).
__device__ __forceinline__ void philox4x32_10(const Params& p, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              uint32_t& w0, uint32_t& w1, uint32_t& w2, uint32_t& w3)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        const uint32_t n0 = hi1 ^ c1 ^ p.k0[r];
        const uint32_t n2 = hi0 ^ c3 ^ p.k1[r];
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    }
    w0 = c0; w1 = c1; w2 = c2; w3 = c3;
}

// d / L (seam ids); a shift when L is a power of two.
__device__ __forceinline__ uint32_t div_L(const Params& p, uint32_t d)
{
    return p.logL >= 0 ? (d >> p.logL) : d / (uint32_t)p.L;
}

// 4 bits (bit j = byte j of a equals byte j of b)
__device__ __forceinline__ uint32_t eq_bytes4(uint32_t a, uint32_t b)
{
    return ((__vcmpeq4(a, b) & 0x08040201u) * 0x01010101u) >> 24;
}

// spread 4 bits to 4 bytes of 0/1
__device__ __forceinline__ uint32_t bits_to_bytes4(uint32_t b)
{
    return ((b & 0xFu) * 0x00204081u) & 0x01010101u;
}

__device__ __forceinline__ uint32_t lanemask_lt()
{
    uint32_t m;
    asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
    return m;
}

// Device-side accumulators at the start of the workspace (zeroed by sw_bind; parts re-zeroed per call).
constexpr int ACC_PARTS = 32;
struct AccPart {                       // one 128-byte line per part: same-address atomics serialise in one L2 slice
    unsigned long long n_active;       // bonds activated by the last sweep / step
    unsigned long long n_clusters;     // roots counted by the last flatten pass
    unsigned long long sat;            // satisfied bonds / sites in state 1 of the configuration the last sweep STARTED from
    unsigned long long minus;          // (counted by k_scan from the spins it reads anyway; q = 2 only for `minus`)
    unsigned long long pad[12];
};
struct Acc {
    AccPart part[ACC_PARTS];           // per-sweep counters: the sum over the parts is the value
    unsigned long long sat;            // observables
    unsigned long long cnt[8];
    unsigned long long cs_nclusters;   // cluster statistics
    unsigned long long cs_max;
    unsigned long long cs_sumsq;
    unsigned long long hist[32];
};
constexpr int WOLFF_RING = 1024;       // per-step |C| slots between host flushes
constexpr int SERIES_RING = 4096;      // sweeps whose (sat, minus) are kept for sw_series_read
struct SeriesEntry { unsigned long long sat, minus; };

}  // namespace swb
