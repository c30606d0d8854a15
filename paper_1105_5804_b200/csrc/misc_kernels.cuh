// misc_kernels.cuh -- support kernels: initialisation (S:8a a8), materialised bond activation (a1, sw_activate),
// energy / magnetisation reduction (a6) and cluster statistics (a9).
#pragma once
#include "common.cuh"

namespace swb {

__device__ __forceinline__ uint32_t store_byte(int q, uint32_t k)
{
    return q == 2 ? (k ? 0xFFu : 0x01u) : k;             // Ising storage: k=0 -> +1, k=1 -> -1
}

// S:8c.8: cold: all k=0; random: k_i = (PHILOX(seed; i>>2, 0, 0, INIT)[i&3] * q) >> 32.  One thread per 4 sites.
__global__ void __launch_bounds__(256)
k_init(const Params p, uint32_t* __restrict__ spins_w, int mode)
{
    const int nw = p.N >> 2;
    for (int i4 = blockIdx.x * blockDim.x + threadIdx.x; i4 < nw; i4 += gridDim.x * blockDim.x) {
        uint32_t k0 = 0, k1 = 0, k2 = 0, k3 = 0;
        if (mode == 1) {
            uint32_t w0, w1, w2, w3;
            philox4x32_10(p, (uint32_t)i4, 0u, 0u, DOM_INIT, w0, w1, w2, w3);
            k0 = __umulhi(w0, (uint32_t)p.q); k1 = __umulhi(w1, (uint32_t)p.q);
            k2 = __umulhi(w2, (uint32_t)p.q); k3 = __umulhi(w3, (uint32_t)p.q);
        }
        spins_w[i4] = store_byte(p.q, k0) | (store_byte(p.q, k1) << 8) | (store_byte(p.q, k2) << 16) |
                      (store_byte(p.q, k3) << 24);
    }
}

// Packed bonds of step t for the current spins (P:70 bond array; S:8c.3-4).  One thread per 16 sites = 4 bytes (N/4 is a
// multiple of 4 because L is), the same draw-to-bit arithmetic as k_scan (scan_kernel.cuh bond_byte).
template <bool ISING>
__global__ void __launch_bounds__(256)
k_activate(const Params p, const uint32_t* __restrict__ spins_w, uint8_t* __restrict__ bonds)
{
    const int L = p.L, Lw = L >> 2, nq = p.N >> 4;
    for (int i16 = blockIdx.x * blockDim.x + threadIdx.x; i16 < nq; i16 += gridDim.x * blockDim.x) {
        uint32_t out = 0;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const int i4 = 4 * i16 + k;
            const int yy = p.logL >= 0 ? (i4 >> (p.logL - 2)) : i4 / Lw, xw = i4 - yy * Lw;
            const uint32_t w = spins_w[i4];
            const uint32_t we = spins_w[yy * Lw + (xw + 1 == Lw ? 0 : xw + 1)];
            const uint32_t wn = spins_w[(yy + 1 == L ? 0 : yy + 1) * Lw + xw];
            // (i>>1) of the first pair of this word = 2 * i4
            const uint32_t d = draw_byte(p, (uint32_t)i4 * 2u, p.t_lo, p.t_hi);
            uint32_t ce, cn;
            out |= bond_byte<ISING>(p, d, w, __funnelshift_r(w, we, 8), wn, ce, cn) << (8 * k);
        }
        reinterpret_cast<uint32_t*>(bonds)[i16] = out;
    }
}

__device__ __forceinline__ unsigned long long warp_sum_u64(unsigned long long v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// S:8a a6 (Eq. 1): satisfied bonds and per-state counts of the current spins, int64 accumulation:
// registers -> warp shuffle -> one 64-bit atomic per warp and quantity.
__global__ void __launch_bounds__(256)
k_observables(const Params p, const uint32_t* __restrict__ spins_w, Acc* __restrict__ acc)
{
    const int L = p.L, Lw = L >> 2;
    unsigned long long sat = 0, cnt[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    // a CTA takes a block of consecutive rows (no index division; the north row of one iteration is the row of the next and
    // comes from the cache); the east word is the next word of the row (periodic)
    const int rows_per = (L + gridDim.x - 1) / gridDim.x;
    const int y_begin = blockIdx.x * rows_per, y_end = min(L, y_begin + rows_per);
    for (int yy = y_begin; yy < y_end; ++yy) {
        const uint32_t* const row = spins_w + (size_t)yy * Lw;
        const uint32_t* const nrow = spins_w + (size_t)(yy + 1 == L ? 0 : yy + 1) * Lw;
        uint32_t s = 0, c = 0;
        auto word = [&](uint32_t w, uint32_t we, uint32_t wn) {
            const uint32_t east = __funnelshift_r(w, we, 8);
            if (p.q == 2) {                              // bytes 0x01 / 0xFF: bit 1 (2) of the xor is set iff the spins differ
                s += 8 - __popc(((w ^ east) & 0x02020202u) | ((w ^ wn) & 0x04040404u));
                c += __popc(w & 0x80808080u);            // bytes equal to -1
            } else {
                s += __popc(eq_bytes4(w, east)) + __popc(eq_bytes4(w, wn));
#pragma unroll
                for (int k = 1; k < 8; ++k)
                    if (k < p.q) cnt[k] += __popc(__vcmpeq4(w, 0x01010101u * k) & 0x01010101u);
            }
        };
        if ((Lw & 3) == 0) {                             // 128-bit loads: 16 sites per thread and iteration
            const int Lv = Lw >> 2;
#pragma unroll 2
            for (int xv = threadIdx.x; xv < Lv; xv += blockDim.x) {
                const uint4 v = reinterpret_cast<const uint4*>(row)[xv];
                const uint4 vn = reinterpret_cast<const uint4*>(nrow)[xv];
                const uint32_t e = row[xv + 1 == Lv ? 0 : 4 * xv + 4];
                word(v.x, v.y, vn.x); word(v.y, v.z, vn.y); word(v.z, v.w, vn.z); word(v.w, e, vn.w);
            }
        } else {
            for (int xw = threadIdx.x; xw < Lw; xw += blockDim.x)
                word(row[xw], row[xw + 1 == Lw ? 0 : xw + 1], nrow[xw]);
        }
        sat += s;
        cnt[1] += c;
    }
    sat = warp_sum_u64(sat);
#pragma unroll
    for (int k = 1; k < 8; ++k) cnt[k] = warp_sum_u64(cnt[k]);
    if ((threadIdx.x & 31) == 0) {
        if (sat) atomicAdd(&acc->sat, sat);
#pragma unroll
        for (int k = 1; k < 8; ++k) if (cnt[k]) atomicAdd(&acc->cnt[k], cnt[k]);
    }
}

// S:8a a9 (P:142 sizes kept in the roots): size[r] += number of sites labelled r.  One CTA per TW x TH strip: the sites of
// a strip carry few distinct labels (one per cluster that enters the strip), so they are first counted in a shared-memory
// hash table (open addressing, as many slots as sites: it cannot overflow) and every distinct label of the strip costs ONE
// global atomic -- the giant cluster at beta_c gets one atomic per strip instead of one per site.  Equal neighbours inside
// a thread's 4 sites are merged before the table is touched.
constexpr int CS_SLOTS = TW * TH;
__global__ void __launch_bounds__(256)
k_cluster_sizes(const Params p, const int* __restrict__ labels, int* __restrict__ size)
{
    __shared__ int s_key[CS_SLOTS];
    __shared__ int s_cnt[CS_SLOTS];
    const int L = p.L;
    const int x0 = blockIdx.x * TW, y0 = blockIdx.y * TH;
    for (int i = threadIdx.x; i < CS_SLOTS; i += blockDim.x) { s_key[i] = -1; s_cnt[i] = 0; }
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
    const int x = x0 + 4 * lane;
    if (x < L) {
        for (int ly = warp; ly < TH && y0 + ly < p.H; ly += nwarp) {
            const int4 v = *reinterpret_cast<const int4*>(labels + (size_t)(y0 + ly) * L + x);
            int lab[4] = {v.x, v.y, v.z, v.w};
            int cnt[4] = {1, 1, 1, 1};
#pragma unroll
            for (int j = 1; j < 4; ++j)
                if (lab[j] == lab[j - 1]) { cnt[j] += cnt[j - 1]; cnt[j - 1] = 0; }
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                if (cnt[j] == 0) continue;
                uint32_t slot = ((uint32_t)lab[j] * 0x9E3779B1u) >> (32 - TW_LOG - TH_LOG);
                while (true) {
                    const int old = atomicCAS(&s_key[slot], -1, lab[j]);
                    if (old == -1 || old == lab[j]) break;
                    slot = (slot + 1) & (CS_SLOTS - 1);
                }
                atomicAdd(&s_cnt[slot], cnt[j]);
            }
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < CS_SLOTS; i += blockDim.x)
        if (s_key[i] >= 0) atomicAdd(&size[s_key[i]], s_cnt[i]);
}

// Statistics over the roots (labels[i] == i): count, maximum, sum of squares, log2-binned histogram.
__global__ void __launch_bounds__(256)
k_cluster_stats(const Params p, const int* __restrict__ labels, const int* __restrict__ size, Acc* __restrict__ acc)
{
    __shared__ unsigned int s_hist[32];                  // per-CTA counts fit 32 bits (native shared-memory atomics)
    __shared__ unsigned long long s_n, s_max, s_sq;
    if (threadIdx.x < 32) s_hist[threadIdx.x] = 0;
    if (threadIdx.x == 0) { s_n = 0; s_max = 0; s_sq = 0; }
    __syncthreads();
    unsigned long long n = 0, mx = 0, sq = 0;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < p.N; i += gridDim.x * blockDim.x) {
        if (labels[i] == i) {
            const unsigned long long s = (unsigned long long)(unsigned)size[i];
            ++n;
            mx = s > mx ? s : mx;
            sq += s * s;
            atomicAdd(&s_hist[31 - __clz((unsigned)s)], 1u);
        }
    }
    n = warp_sum_u64(n);
    sq = warp_sum_u64(sq);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const unsigned long long other = __shfl_xor_sync(0xffffffffu, mx, o);
        mx = other > mx ? other : mx;
    }
    if ((threadIdx.x & 31) == 0) {
        atomicAdd(&s_n, n);
        atomicAdd(&s_sq, sq);
        atomicMax(&s_max, mx);
    }
    __syncthreads();
    if (threadIdx.x < 32 && s_hist[threadIdx.x]) atomicAdd(&acc->hist[threadIdx.x], (unsigned long long)s_hist[threadIdx.x]);
    if (threadIdx.x == 0) {
        if (s_n) atomicAdd(&acc->cs_nclusters, s_n);
        if (s_sq) atomicAdd(&acc->cs_sumsq, s_sq);
        atomicMax(&acc->cs_max, s_max);
    }
}

}  // namespace swb
