// cubic_kernels.cuh -- Swendsen-Wang sweep of the q-state Potts / Ising model on the periodic L x L x L simple cubic lattice
// (S:8f row 2; "hypercubic lattices": in three dimensions every site looks after "three out of six neighbours").
//
// Site i = z L^2 + y L + x owns its bonds to the east (x+1), north (y+1) and up (z+1) neighbour.  Draws (DESIGN.md reading
// 19): u3(i,d,t) = PHILOX(seed; i, t, BOND3)[d], one call per site.  The three steps in three launches:
//   k3_local : bond activation fused with tile-local labelling.  A CTA stages a C3X x C3Y x C3Z tile (32 x 8 x 8 sites) in
//              shared memory: bonds from the spins and Philox, a union-find over the tile's sites with atomicMin hooking on
//              shared-memory int32 (larger root under smaller: a root is the minimum index of its set), then one flatten
//              pass; every site's entry in the labels array becomes the GLOBAL index of its tile-local root.  The 3 bond bits
//              per site go to a byte array (the faces need them; sw_activate returns them).  The energy / magnetisation of
//              the configuration the sweep starts from are counted on the way (a6).
//   k3_faces : cross-tile consolidation (a3): for every active bond that leaves a tile (28 % of the sites own one), the
//              lock-free union by minimum index of label_kernels.cuh (gunite: atomicMin root-to-root hooks, path halving)
//              on the labels array, whose entries are all parent pointers (>= 0, <= own index).
//   k3_final : flatten + flip (a4 + a5): every site chases to the root of its tree (one or two hops), writes the canonical
//              label and takes the state PHILOX(seed; root, t, FLIP) draws; concurrent writes of final labels are roots of
//              the same tree, so a chase that meets one still ends at the right root (same argument as k_final).
// The labels make one HBM round trip as in 2D; per site: spins 1 + bond byte 1 + entry 4 | entry 4 + label 4 + spin 1 = 15 B.
#pragma once
#include "common.cuh"
#include "label_kernels.cuh"

namespace swb {

#ifndef SWB_C3Y
#define SWB_C3Y 8
#endif
#ifndef SWB_C3Z
#define SWB_C3Z 8
#endif
#ifndef SWB_C3CTAS
#define SWB_C3CTAS 8                                     // resident CTAs per SM k3_local is compiled for (32 registers): it is
#endif                                                   // bound by shared-memory latency; 4 CTAs: 0.51 ms at L=256, 8: 0.36
constexpr int C3X = 32, C3Y = SWB_C3Y, C3Z = SWB_C3Z;                // tile: x extent = one 32-byte sector of spins, 128 bytes of labels
constexpr int C3SITES = C3X * C3Y * C3Z;
constexpr int C3THREADS = 256;
constexpr int C3ITEMS = C3SITES / 4 / C3THREADS;         // 32-bit spin words (4 sites) per thread
constexpr uint32_t DOM_BOND3 = 4;
static_assert(C3ITEMS * C3THREADS * 4 == C3SITES, "tile / thread mapping");

// bond bits of the 4 sites of one spin word: byte j of the result = bit 0 east, bit 1 north, bit 2 up of site i0 + j.
// w = the sites' spins, e / n / u = spins of their east / north / up neighbours.  sat = satisfied bonds among the 12.
template <bool ISING>
__device__ __forceinline__ uint32_t bonds3_word(const Params& p, uint32_t i0, uint32_t w, uint32_t e, uint32_t n, uint32_t u,
                                                uint32_t& sat)
{
    // byte-wise equality masks (0xFF where equal); Ising bytes are 0x01 / 0xFF, Potts bytes the state
    const uint32_t qe = __vcmpeq4(w, e), qn = __vcmpeq4(w, n), qu = __vcmpeq4(w, u);
    sat = (__popc(qe) + __popc(qn) + __popc(qu)) >> 3;
    uint32_t out = 0;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        uint32_t d0, d1, d2, d3;
        philox4x32_10(p, i0 + (uint32_t)j, p.t_lo, p.t_hi, DOM_BOND3, d0, d1, d2, d3);
        const uint32_t b = (d0 < p.T ? 1u : 0u) | (d1 < p.T ? 2u : 0u) | (d2 < p.T ? 4u : 0u);
        out |= b << (8 * j);
    }
    return out & ((qe & 0x01010101u) | (qn & 0x02020202u) | (qu & 0x04040404u));
}

// spins of the east neighbours of the 4 sites of word xw in the row that starts at word `row` (Lw words, periodic)
__device__ __forceinline__ uint32_t east_word(const uint32_t* __restrict__ spins_w, size_t row, int xw, int Lw, uint32_t w)
{
    return __funnelshift_r(w, spins_w[row + (xw + 1 == Lw ? 0 : xw + 1)], 8);
}

// find with path halving: a plain store of an ancestor into a non-root entry (roots change only by the atomicMin of
// unite_s; a hook displaced by such a store is re-established by the retry loop there -- DESIGN.md "Concurrency")
__device__ __forceinline__ int find_s(volatile int* lab, int x)
{
    int pp = lab[x];
    while (pp != x) {
        const int gp = lab[pp];
        if (gp == pp) return pp;
        lab[x] = gp;
        x = gp;
        pp = lab[x];
    }
    return x;
}

// lock-free union by minimum index in shared memory (the smem twin of gunite)
__device__ __forceinline__ void unite_s(int* lab, int a, int b)
{
    while (true) {
        a = find_s(lab, a);
        b = find_s(lab, b);
        if (a == b) return;
        if (a < b) { const int t = a; a = b; b = t; }
        const int old = atomicMin(lab + a, b);
        if (old == a) return;
        a = old;
    }
}

struct Tile3 {
    int x0, y0, z0, ex, ey, ez;                          // origin and extent (ragged at the lattice edge)
};
__device__ __forceinline__ Tile3 tile3_of(const Params& p, int t)
{
    Tile3 c;
    const int tx = t % p.n3x, r = t / p.n3x, ty = r % p.n3y, tz = r / p.n3y;
    c.x0 = tx * C3X; c.y0 = ty * C3Y; c.z0 = tz * C3Z;
    c.ex = min(C3X, p.L - c.x0); c.ey = min(C3Y, p.L - c.y0); c.ez = min(C3Z, p.L - c.z0);
    return c;
}

// FROM_BONDS: the bond bytes are an INPUT (sw_label on a cubic handle: `bonds_in`, one byte per site); nothing is drawn,
// no spins are read, no energy is counted.
template <bool ISING, bool FROM_BONDS = false>
__global__ void __launch_bounds__(C3THREADS, SWB_C3CTAS)
k3_local(const Params p, const uint32_t* __restrict__ spins_w, int* __restrict__ prov, uint8_t* __restrict__ bonds,
         Acc* __restrict__ acc, const uint8_t* __restrict__ bonds_in = nullptr)
{
    __shared__ int s_lab[C3SITES];
    __shared__ uint32_t s_bnd[C3SITES / 4];
    const int L = p.L, Lw = L >> 2;
    const Tile3 c = tile3_of(p, blockIdx.x);
    uint32_t nact = 0, nsat = 0, nminus = 0;
    // (1) bonds; every site starts as its own root
#pragma unroll
    for (int k = 0; k < C3ITEMS; ++k) {
        const int item = threadIdx.x + k * C3THREADS;
        const int wx = item % (C3X / 4), r = item / (C3X / 4), ly = r % C3Y, lz = r / C3Y;
        const int l = (lz * C3Y + ly) * C3X + 4 * wx;
        uint32_t b = 0;
        if (4 * wx < c.ex && ly < c.ey && lz < c.ez) {
            const int x = c.x0 + 4 * wx, y = c.y0 + ly, z = c.z0 + lz, xw = x >> 2;
            const size_t row = ((size_t)z * L + y) * Lw;
            const size_t rown = ((size_t)z * L + (y + 1 == L ? 0 : y + 1)) * Lw;
            const size_t rowu = ((size_t)(z + 1 == L ? 0 : z + 1) * L + y) * Lw;
            if (FROM_BONDS) {
                b = reinterpret_cast<const uint32_t*>(bonds_in)[row + xw] & 0x07070707u;
            } else {
                const uint32_t w = spins_w[row + xw];
                uint32_t sat;
                b = bonds3_word<ISING>(p, (uint32_t)((z * L + y) * L + x), w, east_word(spins_w, row, xw, Lw, w), spins_w[rown + xw],
                                       spins_w[rowu + xw], sat);
                nsat += sat;
                if (ISING) nminus += __popc(w & 0x80808080u);
            }
            reinterpret_cast<uint32_t*>(bonds)[row + xw] = b;
            nact += __popc(b);
        }
        s_bnd[l >> 2] = b;
        // the runs along x are labelled right here, without a union: inside the word by the bond bits; across the 8 words of a
        // tile row (8 neighbouring lanes) by a segmented scan -- a word that is one run and linked to its left neighbour
        // passes that neighbour's outgoing root on -- so that every site starts pointing at the first site of its x-run
        const bool e0 = b & 0x00000001u, e1 = b & 0x00000100u, e2 = b & 0x00010000u;
        const bool e3 = (b & 0x01000000u) && 4 * wx + 4 < c.ex;
        const bool link_in = __shfl_up_sync(FULLM, e3, 1, C3X / 4) && wx > 0;
        int val = e2 ? (e1 ? (e0 ? l : l + 1) : l + 2) : l + 3;     // first site of the run that leaves the word to the right
        bool pass = e0 && e1 && e2 && link_in;
#pragma unroll
        for (int d = 1; d < C3X / 4; d <<= 1) {
            const int v = __shfl_up_sync(FULLM, val, d, C3X / 4);
            const bool q = __shfl_up_sync(FULLM, pass, d, C3X / 4);
            if (pass && wx >= d) { val = v; pass = q; }
        }
        const int rin = __shfl_up_sync(FULLM, val, 1, C3X / 4);
        const int f0 = link_in ? rin : l;
        const int l1 = e0 ? f0 : l + 1, l2 = e1 ? l1 : l + 2, l3 = e2 ? l2 : l + 3;
        *reinterpret_cast<int4*>(&s_lab[l]) = make_int4(f0, l1, l2, l3);
    }
    __syncthreads();
    // (2) unions over the bonds that stay inside the tile (the x-runs are labelled already).  North, then up: a thread WALKS
    // a line of sites (north: fixed x and z, y = 0 .. C3Y-1, a warp per plane; up: fixed x and y, z = 0 .. C3Z-1, a warp per row) and carries the root of the set it is in: where the
    // bond to the next site is active that site's tree is united with the carried root (one side of the union needs no
    // find, and sets are joined bottom-up, so the trees stay shallow); where it is not, the walk continues with the next
    // site's root.  Unions are lock-free (other lanes walk the neighbouring lines at the same time): atomicMin hook of the
    // larger root under the smaller.  (One union per bond position of a word, direction by direction: 0.239 ms at L = 256;
    // the walks: see DESIGN.md.)
    static_assert(C3X == 32 && C3THREADS == C3X * C3Y && C3THREADS == C3X * C3Z, "one lane per x, one warp per plane / row");
    const uint8_t* const s_bb = reinterpret_cast<const uint8_t*>(s_bnd);
#pragma unroll
    for (int dir = 1; dir < 3; ++dir) {
        const int lx = threadIdx.x & (C3X - 1), other = threadIdx.x >> 5;        // north: other = z; up: other = y
        const int stride = dir == 1 ? C3X : C3X * C3Y, n = dir == 1 ? c.ey : c.ez;
        int l = (dir == 1 ? other * C3Y * C3X : other * C3X) + lx;
        int root = s_lab[l];
        for (int s = 0; s + 1 < n; ++s) {
            const bool bond = (s_bb[l] >> dir) & 1u;
            l += stride;
            int a = root, b = s_lab[l];
            root = b;
            if (bond) {
                while (true) {                           // unite; the carried root becomes the root of the union
                    a = find_s(s_lab, a);
                    b = find_s(s_lab, b);
                    if (a == b) break;
                    if (a < b) { const int t = a; a = b; b = t; }
                    const int old = atomicMin(s_lab + a, b);
                    if (old == a) { a = b; break; }
                    a = old;
                }
                root = a;
            }
            __syncwarp();
        }
        __syncthreads();
    }
    // (3) every site -> the global index of its tile-local root
#pragma unroll
    for (int k = 0; k < C3ITEMS; ++k) {
        const int item = threadIdx.x + k * C3THREADS;
        const int wx = item % (C3X / 4), r = item / (C3X / 4), ly = r % C3Y, lz = r / C3Y;
        if (4 * wx < c.ex && ly < c.ey && lz < c.ez) {
            const int l = (lz * C3Y + ly) * C3X + 4 * wx;
            int g[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                int rt = l + j, pp = s_lab[rt];          // (read-only chase: the trees are shallow and final)
                while (pp != rt) { rt = pp; pp = s_lab[rt]; }
                const int rx = rt % C3X, rr = rt / C3X, ry = rr % C3Y, rz = rr / C3Y;
                g[j] = ((c.z0 + rz) * L + (c.y0 + ry)) * L + c.x0 + rx;
            }
            *reinterpret_cast<int4*>(prov + ((size_t)((c.z0 + lz) * L + (c.y0 + ly)) * L + c.x0 + 4 * wx)) =
                make_int4(g[0], g[1], g[2], g[3]);
        }
    }
    nact = __reduce_add_sync(FULLM, nact);
    nsat = __reduce_add_sync(FULLM, nsat);
    nminus = __reduce_add_sync(FULLM, nminus);
    if ((threadIdx.x & 31) == 0) {
        AccPart* const part = &acc->part[(blockIdx.x + (threadIdx.x >> 5)) & (ACC_PARTS - 1)];
        if (nact) atomicAdd(&part->n_active, (unsigned long long)nact);
        if (nsat) atomicAdd(&part->sat, (unsigned long long)nsat);
        if (nminus) atomicAdd(&part->minus, (unsigned long long)nminus);
    }
}

// sw_activate on the cubic lattice: the bond bytes of step t for the current spins (one byte per site, bits 0..2)
template <bool ISING>
__global__ void __launch_bounds__(256)
k3_activate(const Params p, const uint32_t* __restrict__ spins_w, uint8_t* __restrict__ bonds)
{
    const int L = p.L, Lw = L >> 2, nw = p.N >> 2;
    for (int i4 = blockIdx.x * blockDim.x + threadIdx.x; i4 < nw; i4 += gridDim.x * blockDim.x) {
        const int xw = i4 % Lw, r = i4 / Lw, y = r % L, z = r / L;
        const size_t row = ((size_t)z * L + y) * Lw;
        const size_t rown = ((size_t)z * L + (y + 1 == L ? 0 : y + 1)) * Lw;
        const size_t rowu = ((size_t)(z + 1 == L ? 0 : z + 1) * L + y) * Lw;
        const uint32_t w = spins_w[i4];
        uint32_t sat;
        reinterpret_cast<uint32_t*>(bonds)[i4] = bonds3_word<ISING>(p, 4u * (uint32_t)i4, w, east_word(spins_w, row, xw, Lw, w),
                                                                    spins_w[rown + xw], spins_w[rowu + xw], sat);
    }
}

// Only the words that own bonds leaving their tile get a thread: ids [0, Wy) the words of the last row of every tile (north
// bonds), [Wy, Wy + Wz) the words of the last plane of every tile (up bonds), then the last site of every tile row (east
// bond).  series != NULL: one thread files the (sat, minus) totals of k3_local under the step counter.
__host__ __device__ inline long long faces3_ids(int L)
{
    const long long Lw = L >> 2, nf = (L + C3Y - 1) / C3Y, nfz = (L + C3Z - 1) / C3Z, nfx = (L + C3X - 1) / C3X;
    return (long long)L * nf * Lw + nfz * (long long)L * Lw + (long long)L * L * nfx;
}
__global__ void __launch_bounds__(256)
k3_faces(const Params p, const uint8_t* __restrict__ bonds, int* prov, const Acc* __restrict__ acc,
         SeriesEntry* __restrict__ series)
{
    if (series != nullptr && blockIdx.x == 0 && threadIdx.x == 0) {
        unsigned long long sat = 0, minus = 0;
        for (int k = 0; k < ACC_PARTS; ++k) { sat += acc->part[k].sat; minus += acc->part[k].minus; }
        SeriesEntry e; e.sat = sat; e.minus = minus;
        series[p.t_lo & (SERIES_RING - 1)] = e;
    }
    const int L = p.L, Lw = L >> 2;
    const int nfy = (L + C3Y - 1) / C3Y, nfz = (L + C3Z - 1) / C3Z, nfx = (L + C3X - 1) / C3X;
    const long long Wy = (long long)L * nfy * Lw, Wz = (long long)nfz * L * Lw;
    long long id = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (id < Wy + Wz) {
        const int d = id < Wy ? 1 : 2;
        int xw, y, z;
        if (d == 1) {
            xw = (int)(id % Lw); const long long r = id / Lw; const int fy = (int)(r % nfy); z = (int)(r / nfy);
            y = min(fy * C3Y + C3Y - 1, L - 1);
        } else {
            id -= Wy;
            xw = (int)(id % Lw); const long long r = id / Lw; y = (int)(r % L); const int fz = (int)(r / L);
            z = min(fz * C3Z + C3Z - 1, L - 1);
        }
        const int i = ((z * L + y) * Lw + xw) * 4;
        const uint32_t b = reinterpret_cast<const uint32_t*>(bonds)[i >> 2] & (0x01010101u << d);
        if (b == 0u) return;
        const int nb = d == 1 ? (y == L - 1 ? i - (L - 1) * L : i + L) : (z == L - 1 ? i - (L - 1) * L * L : i + L * L);
        // the entries of both sides are two 128-bit loads; a site whose two entries equal those of the previous bonded site
        // joins the same two trees (that site does the union)
        const int4 A4 = __ldcg(reinterpret_cast<const int4*>(prov + i)), B4 = __ldcg(reinterpret_cast<const int4*>(prov + nb));
        const int A[4] = {A4.x, A4.y, A4.z, A4.w}, B[4] = {B4.x, B4.y, B4.z, B4.w};
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            if (!(b & (0xFFu << (8 * j)))) continue;
            if (j > 0 && (b & (0xFFu << (8 * (j - 1)))) && A[j] == A[j - 1] && B[j] == B[j - 1]) continue;
            gunite(prov, i + j, nb + j, A[j], B[j]);
        }
        return;
    }
    id -= Wy + Wz;
    if (id < (long long)L * L * nfx) {
        const int fx = (int)(id % nfx); const long long r = id / nfx;         // r = z L + y
        const int x = min(fx * C3X + C3X - 1, L - 1);
        const int i = (int)(r * L) + x;
        if (!(bonds[i] & 1u)) return;
        const int nb = x == L - 1 ? i + 1 - L : i + 1;
        gunite(prov, i, nb, __ldcg(prov + i), __ldcg(prov + nb));
    }
}

// One thread per 4 sites: canonical labels, new spins (flip == false: labels only), number of roots.
// FLIP = false: labels only (sw_label)
template <bool ISING, bool FLIP = true>
__global__ void __launch_bounds__(256)
k3_final(const Params p, int* labels, uint32_t* __restrict__ spins_w, Acc* __restrict__ acc)
{
    const int nw = p.N >> 2;
    unsigned nroots = 0;
    for (int i4 = blockIdx.x * blockDim.x + threadIdx.x; i4 < nw; i4 += gridDim.x * blockDim.x) {
        const int4 v = *reinterpret_cast<const int4*>(labels + 4 * (size_t)i4);
        int rt[4] = {v.x, v.y, v.z, v.w};
        // the four chases in lockstep: four independent loads per round trip (an entry is a parent pointer or, once its
        // thread has been here, the final label: a root of the same tree either way)
        int pp[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) pp[j] = __ldca(labels + rt[j]);
        while ((pp[0] ^ rt[0]) | (pp[1] ^ rt[1]) | (pp[2] ^ rt[2]) | (pp[3] ^ rt[3])) {
#pragma unroll
            for (int j = 0; j < 4; ++j) { rt[j] = pp[j]; pp[j] = __ldca(labels + rt[j]); }
        }
        uint32_t word = 0, state = 0;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            if (FLIP && (j == 0 || rt[j] != rt[j - 1])) state = flip_state(p, rt[j]);
            nroots += rt[j] == 4 * i4 + j;
            word |= (ISING ? (state ? 0xFFu : 0x01u) : state) << (8 * j);
        }
        *reinterpret_cast<int4*>(labels + 4 * (size_t)i4) = make_int4(rt[0], rt[1], rt[2], rt[3]);
        if (FLIP) spins_w[i4] = word;
    }
    nroots = __reduce_add_sync(FULLM, nroots);
    if ((threadIdx.x & 31) == 0 && nroots)
        atomicAdd(&acc->part[(blockIdx.x + (threadIdx.x >> 5)) & (ACC_PARTS - 1)].n_clusters, (unsigned long long)nroots);
}

// a6 of the CURRENT spins on the cubic lattice: satisfied bonds (of 3N) and per-state counts
__global__ void __launch_bounds__(256)
k3_observables(const Params p, const uint32_t* __restrict__ spins_w, Acc* __restrict__ acc)
{
    const int L = p.L, Lw = L >> 2, nw = p.N >> 2;
    unsigned long long sat = 0, cnt[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    for (int i4 = blockIdx.x * blockDim.x + threadIdx.x; i4 < nw; i4 += gridDim.x * blockDim.x) {
        const int xw = i4 % Lw, r = i4 / Lw, y = r % L, z = r / L;
        const size_t row = ((size_t)z * L + y) * Lw;
        const size_t rown = ((size_t)z * L + (y + 1 == L ? 0 : y + 1)) * Lw;
        const size_t rowu = ((size_t)(z + 1 == L ? 0 : z + 1) * L + y) * Lw;
        const uint32_t w = spins_w[i4];
        const uint32_t e = east_word(spins_w, row, xw, Lw, w), n = spins_w[rown + xw], u = spins_w[rowu + xw];
        sat += (__popc(__vcmpeq4(w, e)) + __popc(__vcmpeq4(w, n)) + __popc(__vcmpeq4(w, u))) >> 3;
        if (p.q == 2) {
            cnt[1] += __popc(w & 0x80808080u);
        } else {
#pragma unroll
            for (int k = 1; k < 8; ++k)
                if (k < p.q) cnt[k] += __popc(__vcmpeq4(w, 0x01010101u * k) & 0x01010101u);
        }
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

}  // namespace swb
