// wolff_kernel.cuh -- frontier growth of ONE Wolff cluster ("wave-front" option (b); S:8f.1).
//
// The bond variables are pure functions of (seed, t, site, direction) (S:8c.3), so the cluster of the seed site in the
// bond graph of step t can be grown from the seed, drawing only the bonds that are looked at, and is the same set the
// "decompose everything, flip one cluster" path (k_scan / k_seam / k_final<MODE_WOLFF>) finds: S:8c.9, bit for bit.
//
// One CTA grows the cluster level by level.  A site is claimed by flipping its spin with an atomic on its 32-bit word
// (Ising: a flipped site no longer equals the cluster's orientation s0, so it is never claimed twice: the flip IS the
// visited mark, as in the serial algorithm); claimed sites are appended to a queue in global memory.  Every level costs a
// few dependent global-memory round trips (queue entry -> neighbour spins -> claim), about 2 microseconds, whatever its
// width: the growth is latency bound by the chemical distance of the cluster (~ size^0.6 at beta_c), which is why it only
// pays for small clusters.  After `max_levels` levels with a non-empty frontier the kernel gives up: it restores the
// spins of every claimed site (they are all in the queue; the paper's reset_inclus()) and the host lets the
// labelling path do that step.
#pragma once
#include "common.cuh"

namespace swb {

constexpr int WOLFF_THREADS = 1024;

__device__ __forceinline__ uint32_t bond_draw(const Params& p, uint32_t site, int dir)
{
    uint32_t w0, w1, w2, w3;
    philox4x32_10(p, site >> 1, p.t_lo, p.t_hi, DOM_BOND, w0, w1, w2, w3);
    const uint32_t k = 2u * (site & 1u) + (uint32_t)dir;
    return k == 0 ? w0 : k == 1 ? w1 : k == 2 ? w2 : w3;
}

// Persistent over steps: the kernel performs steps t, t+1, ... (at most nsteps) and stops at the first one whose frontier
// outlives `max_levels`; *n_done = the number of steps completed, size_out[k] = |C| of step t + k.  The host reads n_done,
// lets the labelling path do the step that was given up, and comes back for the rest.
__global__ void __launch_bounds__(WOLFF_THREADS, 1)
k_wolff_front(Params p, uint32_t* spins_w, int* __restrict__ queue, int max_levels, int nsteps,
              unsigned long long* __restrict__ size_out, int* __restrict__ n_done)
{
    __shared__ int s_tail;
    const int L = p.L, N = p.N;
    const int tid = threadIdx.x;
    int step = 0;
    for (; step < nsteps; ++step) {
        uint32_t w0, w1, w2, w3;
        philox4x32_10(p, 0u, p.t_lo, p.t_hi, DOM_WSEED, w0, w1, w2, w3);
        const int i0 = (int)__umulhi(w0, (uint32_t)N);
        __syncthreads();                                 // the previous step's flips are done (and s_tail has been read)
        const uint32_t s0 = (__ldcg(spins_w + (i0 >> 2)) >> (8 * (i0 & 3))) & 0xFFu;   // 0x01 (+1) or 0xFF (-1)
        __syncthreads();                                 // everybody has read the seed's spin before it is flipped
        // claim: s0 -> -s0.  +1 -> -1 sets bits 1..7, -1 -> +1 clears them; the old byte tells whether this thread was first
        auto claim = [&](int j) -> bool {
            const int sh = 8 * (j & 3);
            const uint32_t old = s0 == 0x01u ? atomicOr(spins_w + (j >> 2), 0xFEu << sh)
                                             : atomicAnd(spins_w + (j >> 2), ~(0xFEu << sh));
            return ((old >> sh) & 0xFFu) == s0;
        };
        if (tid == 0) {
            claim(i0);
            queue[0] = i0;
            s_tail = 1;
        }
        __syncthreads();
        int head = 0, level = 0;
        bool gave_up = false;
        while (true) {
            const int tail = s_tail;
            if (head == tail) break;
            if (level == max_levels) { gave_up = true; break; }
            __syncthreads();                             // everybody has read s_tail before it moves
            for (int idx = head + tid; idx < tail; idx += WOLFF_THREADS) {
                const int i = __ldcg(queue + idx);
                const int y = i / L, x = i - y * L;
                const int nb[4] = {x + 1 == L ? i + 1 - L : i + 1,      // east:  bond (i, east)
                                   y + 1 == L ? i + L - N : i + L,      // north: bond (i, north)
                                   x == 0 ? i + L - 1 : i - 1,          // west:  bond (west, east)
                                   y == 0 ? i + N - L : i - L};         // south: bond (south, north)
                uint32_t sp[4];
#pragma unroll
                for (int k = 0; k < 4; ++k) sp[k] = (__ldcg(spins_w + (nb[k] >> 2)) >> (8 * (nb[k] & 3))) & 0xFFu;
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    if (sp[k] != s0) continue;           // other orientation, or claimed already
                    const uint32_t u = k < 2 ? bond_draw(p, (uint32_t)i, k) : bond_draw(p, (uint32_t)nb[k], k - 2);
                    if (u < p.T && claim(nb[k])) queue[atomicAdd(&s_tail, 1)] = nb[k];
                }
            }
            __syncthreads();                             // the level's appends (shared counter, global queue) are visible
            head = tail;
            ++level;
        }
        const int total = s_tail;
        if (gave_up) {                                   // restore every claimed site: -s0 -> s0
            for (int idx = tid; idx < total; idx += WOLFF_THREADS) {
                const int j = __ldcg(queue + idx), sh = 8 * (j & 3);
                if (s0 == 0x01u) atomicAnd(spins_w + (j >> 2), ~(0xFEu << sh)); else atomicOr(spins_w + (j >> 2), 0xFEu << sh);
            }
            break;
        }
        if (tid == 0) size_out[step] = (unsigned long long)total;
        if (++p.t_lo == 0u) ++p.t_hi;                    // next step counter
    }
    if (tid == 0) *n_done = step;
}

}  // namespace swb
