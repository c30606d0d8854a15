// paper_kernels.cuh -- the PAPER'S OWN labelling pipeline re-implemented on sm_100a as an ablation baseline (S:8f row 4):
//   kp_selflabel : tile-local SELF-LABELLING (kernel local_selflabel_small(): one spin per thread, B <= 32): the
//                  labels of a B x B tile sit in shared memory; in every pass a site and its east / north neighbour, if
//                  joined by an active bond, take the minimum of their two labels; passes repeat until __syncthreads_or sees
//                  no re-labelling event (n_B ~ B^{d_min} passes at criticality, Eq. 11).  Result: "complete path
//                  compression": every site holds the index of the minimum site of its tile-local cluster.
//   kp_relax     : tile consolidation by LABEL RELAXATION (kernels prepare_relax() / relax_multithread()): for every
//                  active bond that crosses a tile boundary the labels of the two local roots are set to their minimum;
//                  iterations repeat until nothing changes, the stopping criterion being read by the host between launches
//                  (P:198); n_relax ~ (L/B)^{d_min} (Eq. 13).
//   kp_sew       : tile consolidation by HIERARCHICAL SEWING: level k sews 2 x 2 tiles of size 2^{k-1} B with one
//                  thread block per group; the two horizontal seams by two threads, then the vertical seam by one;
//                  log2(L/B) levels, then the periodic wrap bonds "in an additional step".  Bond insertion is union /
//                  find; the paper balances by (fake) size, here the larger ROOT INDEX goes under the smaller (DESIGN.md reading
//                  7: the canonical root is the minimum site index), which adds at most one level per generation.
//   kp_flatten   : every site takes the label of the root of its tree (the find of the paper's flip kernel).
// One deliberate deviation: the paper's self-labelling and relaxation write the minimum with plain stores and accept lost
// updates ("atomics ... slow down the code"); shared-/global-memory atomicMin is native here and makes every label
// monotone, so it is used.  All three produce the canonical labelling (minimum site index), compared bit for bit with the
// oracle; what is measured is what the paper's design costs on a B200 next to k_scan / k_seam / k_final.
#pragma once
#include "common.cuh"

namespace swb {

__device__ __forceinline__ uint32_t bond_code(const uint8_t* __restrict__ packed, int i)
{
    return (packed[i >> 2] >> (2 * (i & 3))) & 3u;       // bit 0 east, bit 1 north
}

// One CTA per B x B tile, one thread per site.  pass_max: the largest number of passes any tile needed.
template <int B>
__global__ void __launch_bounds__(B * B)
kp_selflabel(int L, const uint8_t* __restrict__ packed, int* __restrict__ labels, int* __restrict__ rlab, int* __restrict__ pass_max)
{
    __shared__ int s_lab[B * B];
    const int lx = threadIdx.x % B, ly = threadIdx.x / B, l = threadIdx.x;
    const int x = blockIdx.x * B + lx, y = blockIdx.y * B + ly, i = y * L + x;
    const uint32_t c = bond_code(packed, i);
    const bool e = (c & 1u) && lx + 1 < B, n = (c & 2u) && ly + 1 < B;      // bonds that stay inside the tile
    s_lab[l] = l;
    __syncthreads();
    int passes = 0;
    int changed;
    do {
        changed = 0;
        if (e) {
            const int a = s_lab[l], b = s_lab[l + 1];
            if (a != b) { const int m = min(a, b); atomicMin(&s_lab[l], m); atomicMin(&s_lab[l + 1], m); changed = 1; }
        }
        if (n) {
            const int a = s_lab[l], b = s_lab[l + B];
            if (a != b) { const int m = min(a, b); atomicMin(&s_lab[l], m); atomicMin(&s_lab[l + B], m); changed = 1; }
        }
        ++passes;
    } while (__syncthreads_or(changed));
    const int r = s_lab[l];
    labels[i] = (blockIdx.y * B + r / B) * L + blockIdx.x * B + r % B;
    if (r == l) rlab[i] = i;                             // the label of a local root (relaxation works on these)
    if (threadIdx.x == 0) atomicMax(pass_max, passes);
}

// the two ends of the boundary-crossing bond owned by site i, or false.  dir 0: east bond of the last column of a tile,
// dir 1: north bond of the last row of a tile (periodic)
__device__ __forceinline__ bool crossing_bond(int L, int B, const uint8_t* __restrict__ packed, int x, int y, int dir, int& i, int& j)
{
    i = y * L + x;
    if (!((bond_code(packed, i) >> dir) & 1u)) return false;
    j = dir == 0 ? y * L + (x + 1 == L ? 0 : x + 1) : (y + 1 == L ? 0 : y + 1) * L + x;
    return true;
}

// One relaxation iteration over all 2 (L/B) L boundary bonds: thread id -> (dir, tile line, position along the line).
// labels[i] = local root of site i (fixed); rlab[r] = current label of local root r (Fig. 5: "the local root labels are
// transmitted to neighbouring tiles, who change their local labels to the minimum of their own and the received labels").
__global__ void __launch_bounds__(256)
kp_relax(int L, int B, const uint8_t* __restrict__ packed, const int* __restrict__ labels, int* rlab, int* __restrict__ changed)
{
    const int nline = L / B, per_dir = nline * L;
    int any = 0;
    for (int id = blockIdx.x * blockDim.x + threadIdx.x; id < 2 * per_dir; id += gridDim.x * blockDim.x) {
        const int dir = id / per_dir, r = id - dir * per_dir, line = r / L, pos = r - line * L;
        const int x = dir == 0 ? line * B + B - 1 : pos, y = dir == 0 ? pos : line * B + B - 1;
        int i, j;
        if (!crossing_bond(L, B, packed, x, y, dir, i, j)) continue;
        const int ri = labels[i], rj = labels[j];
        const int la = __ldcg(rlab + ri), lb = __ldcg(rlab + rj);
        if (la == lb) continue;
        const int m = min(la, lb);
        if (la > m) atomicMin(rlab + ri, m);
        if (lb > m) atomicMin(rlab + rj, m);
        any = 1;
    }
    if (__syncthreads_or(any) && threadIdx.x == 0) *changed = 1;
}

__device__ __forceinline__ int pfind(const int* lab, int x)
{
    int pp = lab[x];
    while (pp != x) { x = pp; pp = lab[x]; }
    return x;
}
__device__ __forceinline__ void psew(int* lab, int i, int j)
{
    const int a = pfind(lab, i), b = pfind(lab, j);
    if (a == b) return;
    if (a < b) lab[b] = a; else lab[a] = b;
}

// Level with tiles of size Bk: one block per 2 x 2 group.  Threads 0 and 1 close the horizontal seam of the left and the
// right column of the group (north bonds of the last row of the lower tiles), then thread 0 closes the vertical seam (east
// bonds of the last column of the two left tiles).  Different groups touch disjoint trees: plain loads and stores.
__global__ void __launch_bounds__(32)
kp_sew(int L, int Bk, const uint8_t* __restrict__ packed, int* labels)
{
    const int gx = blockIdx.x * 2 * Bk, gy = blockIdx.y * 2 * Bk;
    if (threadIdx.x < 2) {
        const int y = gy + Bk - 1;
        for (int x = gx + threadIdx.x * Bk; x < gx + (threadIdx.x + 1) * Bk; ++x) {
            int i, j;
            if (crossing_bond(L, Bk, packed, x, y, 1, i, j)) psew(labels, i, j);
        }
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        const int x = gx + Bk - 1;
        for (int y = gy; y < gy + 2 * Bk; ++y) {
            int i, j;
            if (crossing_bond(L, Bk, packed, x, y, 0, i, j)) psew(labels, i, j);
        }
    }
}

// the bonds that wrap around the lattice, "in an additional step": one thread
__global__ void kp_sew_wrap(int L, const uint8_t* __restrict__ packed, int* labels)
{
    if (blockIdx.x != 0 || threadIdx.x != 0) return;
    for (int x = 0; x < L; ++x) { int i, j; if (crossing_bond(L, L, packed, x, L - 1, 1, i, j)) psew(labels, i, j); }
    for (int y = 0; y < L; ++y) { int i, j; if (crossing_bond(L, L, packed, L - 1, y, 0, i, j)) psew(labels, i, j); }
}

// After relaxation: every site takes the label its local root has converged to.
__global__ void __launch_bounds__(256)
kp_flatten_relax(int N, int* labels, const int* __restrict__ rlab, unsigned long long* __restrict__ n_clusters)
{
    unsigned n = 0;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < N; i += gridDim.x * blockDim.x) {
        const int v = rlab[labels[i]];
        labels[i] = v;
        n += v == i;
    }
    n = __reduce_add_sync(0xffffffffu, n);
    if ((threadIdx.x & 31) == 0 && n) atomicAdd(n_clusters, (unsigned long long)n);
}

// After sewing: a chase to the root of the tree.  Final labels written concurrently are roots of the same tree.
__global__ void __launch_bounds__(256)
kp_flatten(int N, int* labels, unsigned long long* __restrict__ n_clusters)
{
    unsigned n = 0;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < N; i += gridDim.x * blockDim.x) {
        int x = i, pp = __ldcg(labels + x);
        while (pp != x) { x = pp; pp = __ldcg(labels + x); }
        labels[i] = x;
        n += x == i;
    }
    n = __reduce_add_sync(0xffffffffu, n);
    if ((threadIdx.x & 31) == 0 && n) atomicAdd(n_clusters, (unsigned long long)n);
}

}  // namespace swb
