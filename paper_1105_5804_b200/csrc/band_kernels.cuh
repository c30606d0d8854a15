// band_kernels.cuh -- multi-GPU Swendsen-Wang by ROW BANDS with one seam exchange per sweep (S:8e, S:8f row 3; the paper's own
// proposal is label relaxation between GPUs over MPI).
//
// Rank r of G works on the strip rows [ty0, ty0 + nband) of the SAME L x L index space: every array is allocated at full
// size on every rank (1.25 GiB at L = 16384 of 180 GB), so site indices, Philox counters and labels are global and the
// single-GPU kernels run unchanged on a band (k_scan / k_final take their strip row from blockIdx.y + ty0; k_seam<BAND> unites
// the seams inside the band).  What crosses ranks per sweep:
//   before the sweep : the spins of the first row above the band (L bytes from the rank above; the top band wraps to row 0),
//                      copied into that row of the local spin array -- k_scan reads it as the north halo;
//   after k_seam     : k_band_resolve replaces the strip-local roots on the band's two outer rows (edge arrays: rootN of its
//                      last row, rootS of its first row) by the roots of the BAND's forest; these 2 L int32 (128 KiB at
//                      L = 16384) are all-gathered into the same rows of every rank's edge arrays;
//   then, redundantly on every rank: k_band_init makes every gathered root that lies outside the band a root of the local
//                      labels array (entry = own index: the array is full size, the entry exists), and k_band_cross unites
//                      the G cross-band seams with the lock-free union of the single-GPU seam pass (gunite).  The local
//                      forest now contains the other bands' roots wherever a cluster of this band reaches them, its roots are
//                      the global minimum site indices, and k_final flattens and flips the band as on one GPU: the cluster
//                      draw is keyed by the global root, so no spin state crosses ranks (the paper's objection that "cluster
//                      roots are scattered", does not arise).
// Observables: k_scan's and k_final's per-sweep counters cover the band; the host binding all-reduces them.
#pragma once
#include "common.cuh"
#include "label_kernels.cuh"

namespace swb {

__device__ __forceinline__ bool in_band(const Params& p, int site)
{
    const int tr = (int)div_L(p, (uint32_t)site) >> TH_LOG;
    return tr >= p.ty0 && tr < p.ty0 + p.nband;
}

// rows of the edge arrays that belong to the outer seams of band b (uniform bands of nband strip rows):
// rootN: edgeA[nE + (last strip row of b) * L + x]; rootS: edgeB[nE + (first strip row of b) * L + x]
__device__ __forceinline__ int band_top_row(const Params& p, int b) { return (b + 1) * p.nband - 1; }

// my two outer rows: strip-local roots -> roots of the band's forest (after k_seam<BAND>)
__global__ void __launch_bounds__(256)
k_band_resolve(const Params p, int* __restrict__ edgeA, int* __restrict__ edgeB, const int* prov)
{
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    if (x >= p.L) return;
    const int nE = p.ntx * p.L;
    int* const a = edgeA + nE + (p.ty0 + p.nband - 1) * p.L + x;
    int* const b = edgeB + nE + p.ty0 * p.L + x;
    const int ra = *a, rb = *b;
    if (ra >= 0) *a = gfind(prov, ra);
    *b = gfind(prov, rb);
}

// every gathered root outside my band becomes a root of my labels array
__global__ void __launch_bounds__(256)
k_band_init(const Params p, const int* __restrict__ edgeA, const int* __restrict__ edgeB, int* prov, int nbands)
{
    const int id = blockIdx.x * blockDim.x + threadIdx.x;
    if (id >= nbands * p.L) return;
    const int b = id / p.L, x = id - b * p.L, nE = p.ntx * p.L;
    const int ra = edgeA[nE + band_top_row(p, b) * p.L + x], rb = edgeB[nE + b * p.nband * p.L + x];
    if (ra >= 0 && !in_band(p, ra)) prov[ra] = ra;
    if (!in_band(p, rb)) prov[rb] = rb;
}

// the north seams on top of every band (the last one wraps to row 0): one seam site per thread
__global__ void __launch_bounds__(256)
k_band_cross(const Params p, const int* __restrict__ edgeA, const int* __restrict__ edgeB, int* prov, int nbands)
{
    const int id = blockIdx.x * blockDim.x + threadIdx.x;
    int ra = -1, rb = -1;
    if (id < nbands * p.L) {
        const int b = id / p.L, x = id - b * p.L, nE = p.ntx * p.L;
        ra = edgeA[nE + band_top_row(p, b) * p.L + x];
        rb = edgeB[nE + (b + 1 == nbands ? 0 : (b + 1) * p.nband) * p.L + x];
    }
    if (seam_todo(ra, rb)) gunite(prov, ra, rb, __ldcg(prov + ra), __ldcg(prov + rb));
}

}  // namespace swb
