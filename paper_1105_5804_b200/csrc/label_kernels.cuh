// label_kernels.cuh -- the Swendsen-Wang hot path (S:8a rows a1-a5, a7):
//   k_local   : bond activation (P:53 step 1, Eq. 7) fused with tile-local labelling in shared memory
//   k_seam    : cross-tile consolidation as ONE concurrent union-find pass over the seam bonds
//   k_seamfix : path compression of the seam roots so that every provisional label is at most 2 hops from its root
//   k_final   : flatten to canonical labels + cluster flip (P:55 step 3) / Wolff flip / label only
// Design notes and the differences from the paper's kernels (self-labelling, hierarchical sewing) are in DESIGN.md.
#pragma once
#include "common.cuh"

namespace swb {

// ------------------------------------------------------------------------------------------------ union-find
// Lock-free union by minimum index on a parent array (shared or global memory).  Invariant: parent[x] <= x, and
// parent[x] only ever changes to a smaller index of the same (growing) set, so a stale read is still an ancestor.
template <typename Ptr>
__device__ __forceinline__ int uf_find(Ptr parent, int x)
{
    int p = parent[x];
    while (p != x) { x = p; p = parent[x]; }
    return x;
}

// find with path halving: every second node on the path is re-pointed at its grandparent.  The plain store races
// with other finds and with atomicMin hooks; it only ever writes an ancestor of x, so the forest stays valid.
__device__ __forceinline__ int uf_find_halve(volatile int* parent, int x)
{
    int p = parent[x];
    while (p != x) {
        const int gp = parent[p];
        if (gp == p) return p;
        parent[x] = gp;
        x = gp;
        p = parent[x];
    }
    return x;
}

__device__ __forceinline__ void uf_unite_shared(int* parent, int a, int b)
{
    volatile int* vp = parent;
    while (true) {
        a = uf_find_halve(vp, a);
        b = uf_find_halve(vp, b);
        if (a == b) return;
        if (a < b) { int t = a; a = b; b = t; }          // a > b: hook a under b
        const int old = atomicMin(&parent[a], b);
        if (old == a) return;                            // a was a root and now points to b
        a = old;                                         // a had been hooked meanwhile: parent[a] = min(old,b); join old and b
    }
}

struct LdCg {                                            // global loads that bypass the (incoherent) L1
    const int* p;
    __device__ __forceinline__ int operator[](int i) const { return __ldcg(p + i); }
};

__device__ __forceinline__ void uf_unite_global(int* parent, int a, int b)
{
    LdCg vp{parent};
    while (true) {
        a = uf_find(vp, a);
        b = uf_find(vp, b);
        if (a == b) return;
        if (a < b) { int t = a; a = b; b = t; }
        const int old = atomicMin(&parent[a], b);
        if (old == a) return;
        a = old;
    }
}

// ------------------------------------------------------------------------------------------------ k_local
// One CTA per TW x TH tile.  FROM_BONDS=false: read spins, draw bonds (a1).  FROM_BONDS=true: read packed bonds
// (sw_label).  Writes provisional labels (global index of the tile-local root = minimum index inside the tile),
// the bonds that cross the tile's east / north edge into seamE / seamN (one byte per seam site), and adds the
// number of active bonds to acc->n_active.
template <bool FROM_BONDS>
__global__ void __launch_bounds__(NTHREADS)
k_local(const Params p, const uint32_t* __restrict__ spins_w, const uint8_t* __restrict__ bonds_in,
        int* __restrict__ labels, uint8_t* __restrict__ seamE, uint8_t* __restrict__ seamN, Acc* __restrict__ acc)
{
    __shared__ __align__(16) int parent[TW * TH];
    __shared__ uint32_t s_efirst[NWARPS][32];            // east bonds of every warp's first row (4 bits per lane)
    constexpr int R = ROWS_PER_WARP;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int L = p.L;
    const int x0 = blockIdx.x * TW, y0 = blockIdx.y * TH;
    const int tw_eff = min(TW, L - x0), th_eff = min(TH, L - y0);
    const int x = x0 + 4 * lane;
    const bool colv = 4 * lane < tw_eff;
    const int last_lane = (tw_eff >> 2) - 1;             // lane that owns the tile's last column
    const int ly0 = warp * R;

    uint32_t ebits = 0, nbits = 0;                       // 4 bits per row r at bit 4r
    int nact = 0;

    if (!FROM_BONDS) {
        const int Lw = L >> 2;                           // words per row
        // my word in rows ly0 .. ly0+R (the last one is only the north neighbour of row R-1)
        uint32_t w[R + 1];
#pragma unroll
        for (int r = 0; r <= R; ++r) {
            const int y = y0 + ly0 + r;                  // y == L: periodic wrap, north neighbour of the last row
            w[r] = (colv && y <= L) ? spins_w[(size_t)(y == L ? 0 : y) * Lw + (x >> 2)] : 0u;
        }
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int y = y0 + ly0 + r;
            const bool rowv = y < L;                     // warp-uniform
            uint32_t wnext = __shfl_down_sync(0xffffffffu, w[r], 1);
            if (rowv && colv && lane == last_lane) {     // east halo: first word of the next tile (periodic)
                const int xe = (x + 4 == L) ? 0 : x + 4;
                wnext = spins_w[(size_t)y * Lw + (xe >> 2)];
            }
            if (rowv && colv) {
                const uint32_t east = __funnelshift_r(w[r], wnext, 8);
                const uint32_t eqe = eq_bytes4(w[r], east);
                const uint32_t eqn = eq_bytes4(w[r], w[r + 1]);
                const uint32_t c0 = (uint32_t)(y * L + x) >> 1;
                uint32_t a0, a1, a2, a3, b0, b1, b2, b3;
                philox4x32_10(p, c0, p.t_lo, p.t_hi, DOM_BOND, a0, a1, a2, a3);
                philox4x32_10(p, c0 + 1, p.t_lo, p.t_hi, DOM_BOND, b0, b1, b2, b3);
                const uint32_t de = (a0 < p.T) | ((a2 < p.T) << 1) | ((b0 < p.T) << 2) | ((b2 < p.T) << 3);
                const uint32_t dn = (a1 < p.T) | ((a3 < p.T) << 1) | ((b1 < p.T) << 2) | ((b3 < p.T) << 3);
                const uint32_t e4 = eqe & de, n4 = eqn & dn;
                nact += __popc(e4) + __popc(n4);
                ebits |= e4 << (4 * r);
                nbits |= n4 << (4 * r);
            }
        }
    } else {
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int y = y0 + ly0 + r;
            if (y < L && colv) {
                const uint32_t b = bonds_in[((size_t)y * L + x) >> 2];
                const uint32_t e4 = (b & 1) | ((b >> 1) & 2) | ((b >> 2) & 4) | ((b >> 3) & 8);
                const uint32_t n4 = ((b >> 1) & 1) | ((b >> 2) & 2) | ((b >> 3) & 4) | ((b >> 4) & 8);
                ebits |= e4 << (4 * r);
                nbits |= n4 << (4 * r);
            }
        }
    }

    // bonds crossing the tile edge go to the seam arrays and are removed from the local masks
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int ly = ly0 + r, y = y0 + ly;
        if (y < L && colv) {
            if (lane == last_lane) {
                seamE[(size_t)blockIdx.x * L + y] = (uint8_t)((ebits >> (4 * r + 3)) & 1u);
                ebits &= ~(8u << (4 * r));
            }
            if (ly == th_eff - 1) {
                *reinterpret_cast<uint32_t*>(seamN + (size_t)blockIdx.y * L + x) = bits_to_bytes4(nbits >> (4 * r));
                nbits &= ~(0xFu << (4 * r));
            }
        }
    }

    s_efirst[warp][lane] = ebits & 0xFu;

    // run starts: every site points to the first site of its horizontal run inside the tile (HA4-style run labelling)
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int ly = ly0 + r;
        const bool rowv = y0 + ly < L;                   // warp-uniform
        const uint32_t e4 = (ebits >> (4 * r)) & 0xFu;
        const uint32_t nf = __ballot_sync(0xffffffffu, e4 != 0xFu);
        const uint32_t hz = ~e4 & 0xFu;                  // broken east bonds inside my group
        const int brk = 4 * lane + (32 - __clz(hz));     // first site after my last broken bond (valid if hz != 0)
        const uint32_t cand = nf & lanemask_lt();
        const int src = cand ? 31 - __clz(cand) : 0;
        int sin = __shfl_sync(0xffffffffu, brk, src);    // start of the run that enters my group from the west
        if (!cand) sin = 0;
        if (rowv && colv) {
            int4 s;
            const int base = ly * TW;
            uint32_t z;
            s.x = base + sin;
            z = hz & 1u; s.y = base + (z ? 4 * lane + (32 - __clz(z)) : sin);
            z = hz & 3u; s.z = base + (z ? 4 * lane + (32 - __clz(z)) : sin);
            z = hz & 7u; s.w = base + (z ? 4 * lane + (32 - __clz(z)) : sin);
            *reinterpret_cast<int4*>(&parent[base + 4 * lane]) = s;
        }
    }
    __syncthreads();

    // north bonds: unite (x,y) with (x,y+1).  A bond is skipped when the site to its west has a north bond too and
    // both horizontal bonds between the two columns are active (it joins the same two runs).  The remaining bonds
    // of the thread's 8 rows are one 32-bit work mask, so lanes stay busy as long as they have any union left.
    {
        const uint32_t e_next = (warp + 1 < NWARPS) ? s_efirst[warp + 1][lane] : 0u;
        const uint32_t e_up = (ebits >> 4) | (e_next << 28);          // east bonds of the row above each row
        const uint32_t X = nbits & ebits & e_up;
        uint32_t Xprev = __shfl_up_sync(0xffffffffu, X, 1);
        if (lane == 0) Xprev = 0;
        const uint32_t redundant = ((X << 1) & 0xEEEEEEEEu) | ((Xprev >> 3) & 0x11111111u);
        uint32_t U = nbits & ~redundant;
        while (U) {
            const int b = __ffs(U) - 1;
            U &= U - 1;
            const int idx = (ly0 + (b >> 2)) * TW + 4 * lane + (b & 3);
            uf_unite_shared(parent, idx, idx + TW);
        }
    }
    __syncthreads();

    // resolve every site to its tile-local root and write the root's global index
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int ly = ly0 + r, y = y0 + ly;
        if (y < L && colv) {
            const int4 a = *reinterpret_cast<const int4*>(&parent[ly * TW + 4 * lane]);
            int4 g;
            volatile int* vp = parent;
            int root = uf_find_halve(vp, a.x);
            g.x = (y0 + root / TW) * L + x0 + (root % TW);
            if (a.y != a.x) root = uf_find_halve(vp, a.y);
            g.y = (y0 + root / TW) * L + x0 + (root % TW);
            if (a.z != a.y) root = uf_find_halve(vp, a.z);
            g.z = (y0 + root / TW) * L + x0 + (root % TW);
            if (a.w != a.z) root = uf_find_halve(vp, a.w);
            g.w = (y0 + root / TW) * L + x0 + (root % TW);
            *reinterpret_cast<int4*>(labels + (size_t)y * L + x) = g;
        }
    }

    if (!FROM_BONDS) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) nact += __shfl_xor_sync(0xffffffffu, nact, o);
        if (lane == 0 && nact) atomicAdd(&acc->n_active, (unsigned long long)nact);
    }
}

// ------------------------------------------------------------------------------------------------ seams
// Seam site id -> the two end sites of its crossing bond.  ids [0, ntx*L): east seams (tile column tc, row y);
// ids [ntx*L, (ntx+nty)*L): north seams (tile row tr, column x).
__device__ __forceinline__ void seam_sites(const Params& p, int id, int& a, int& b)
{
    const int L = p.L;
    const int nE = p.ntx * L;
    if (id < nE) {
        const int tc = div_L(p, (uint32_t)id), y = id - tc * L;
        const int xs = min((tc + 1) * TW, L) - 1;
        a = y * L + xs;
        b = y * L + (xs + 1 == L ? 0 : xs + 1);
    } else {
        const int k = id - nE;
        const int tr = div_L(p, (uint32_t)k), x = k - tr * L;
        const int ys = min((tr + 1) * TH, L) - 1;
        a = ys * L + x;
        b = (ys + 1 == L ? 0 : ys + 1) * L + x;
    }
}

// One thread per seam site: if its crossing bond is active, unite the provisional roots of its two ends.
// `seam` is seamE followed by seamN (contiguous).
__global__ void __launch_bounds__(256)
k_seam(const Params p, const uint8_t* __restrict__ seam, int* __restrict__ labels)
{
    const int nseam = (p.ntx + p.nty) * p.L;
    const int id = blockIdx.x * blockDim.x + threadIdx.x;
    const bool on = id < nseam && seam[id];
    int ra = -1, rb = -1;
    if (on) {
        int a, b;
        seam_sites(p, id, a, b);
        ra = __ldcg(labels + a);
        rb = __ldcg(labels + b);
    }
    // the previous seam site joins the same two provisional clusters: skip (its thread does the union)
    const int pa = __shfl_up_sync(0xffffffffu, ra, 1), pb = __shfl_up_sync(0xffffffffu, rb, 1);
    const bool dup = (threadIdx.x & 31) != 0 && pa == ra && pb == rb;
    if (on && !dup) uf_unite_global(labels, ra, rb);
}

// After k_seam: for both ends of every active seam bond, point the site and its provisional root straight at the
// final root.  Every provisional root that was hooked has such a site in its tile-local cluster, so afterwards
// root(i) = labels[labels[i]] for every site i (2-hop guarantee used by k_final).
__global__ void __launch_bounds__(256)
k_seamfix(const Params p, const uint8_t* __restrict__ seam, int* __restrict__ labels)
{
    const int nseam = (p.ntx + p.nty) * p.L;
    const int id = blockIdx.x * blockDim.x + threadIdx.x;
    if (id >= nseam || !seam[id]) return;
    int s[2];
    seam_sites(p, id, s[0], s[1]);
    LdCg vp{labels};
#pragma unroll
    for (int e = 0; e < 2; ++e) {
        const int x1 = vp[s[e]];
        const int g = uf_find(vp, x1);
        if (x1 != g) {                                   // every writer stores the same final root: benign
            labels[x1] = g;
            labels[s[e]] = g;
        }
    }
}

// ------------------------------------------------------------------------------------------------ k_final
enum { MODE_SW = 0, MODE_WOLFF = 1, MODE_LABEL = 2 };

__device__ __forceinline__ uint32_t flip_state(const Params& p, int root)
{
    uint32_t w0, w1, w2, w3;
    philox4x32_10(p, (uint32_t)root, p.t_lo, p.t_hi, DOM_FLIP, w0, w1, w2, w3);
    return __umulhi(w0, (uint32_t)p.q);                  // uniform state in [0,q)  (S:8c.6)
}

// Shared memory of k_final (dynamic, opt-in above 48 KB): the tile's provisional labels, one state byte per site
// (only written at "anchor" sites) and the compacted list of anchor sites.
struct FinalSmem {
    int      S[TW * TH];
    uint16_t list[TW * TH];
    uint8_t  st[TW * TH];
    int      nlist;
};

// tile-local index of global site v, or -1 if v lies outside the (possibly ragged) tile
__device__ __forceinline__ int tile_local(const Params& p, int v, int base, int tw_eff, int th_eff)
{
    if (v < base) return -1;
    const uint32_t d = (uint32_t)(v - base);
    const uint32_t dy = div_L(p, d), dx = d - dy * (uint32_t)p.L;
    return (dx < (uint32_t)tw_eff && dy < (uint32_t)th_eff) ? (int)(dy * TW + dx) : -1;
}

// One CTA per tile: canonical labels (root of every site) + the new spins.
//   MODE_SW    : s_i = state drawn for the root (assign, P:55 step 3)
//   MODE_WOLFF : s_i = -s_i iff root(i) == root(seed site i0); adds |C| to *wolff_size
//   MODE_LABEL : labels only
// After k_seamfix, root(i) = labels[labels[i]], and the second hop stays inside the tile unless labels[i] already is
// the root.  "Anchor" sites are those whose own label is the final root (roots themselves, and sites pointing out
// of the tile); only they draw a Philox state (compacted, one draw per anchor), every other site copies the state
// of the anchor it resolves to through shared memory.
template <int MODE>
__global__ void __launch_bounds__(NTHREADS, 4)
k_final(const Params p, int* __restrict__ labels, uint32_t* __restrict__ spins_w, Acc* __restrict__ acc,
        unsigned long long* __restrict__ wolff_size)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    FinalSmem& sm = *reinterpret_cast<FinalSmem*>(smem_raw);
    constexpr int R = ROWS_PER_WARP;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int L = p.L;
    const int x0 = blockIdx.x * TW, y0 = blockIdx.y * TH;
    const int tw_eff = min(TW, L - x0), th_eff = min(TH, L - y0);
    const int x = x0 + 4 * lane;
    const bool colv = 4 * lane < tw_eff;
    const int ly0 = warp * R;
    const int base = y0 * L + x0;

    int r0 = -1;
    if (MODE == MODE_WOLFF) {
        uint32_t w0, w1, w2, w3;
        philox4x32_10(p, 0u, p.t_lo, p.t_hi, DOM_WSEED, w0, w1, w2, w3);
        const int i0 = (int)__umulhi(w0, (uint32_t)p.N);
        r0 = __ldcg(labels + __ldcg(labels + i0));       // 2-hop guarantee; stable under concurrent k_final writes
    }
    if (MODE == MODE_SW && threadIdx.x == 0) sm.nlist = 0;

    uint32_t anchor = 0;                                 // bit 4r+j: my site (row r, column j) is an anchor
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int ly = ly0 + r, y = y0 + ly;
        if (y < L && colv) {
            const int4 v = *reinterpret_cast<const int4*>(labels + (size_t)y * L + x);
            *reinterpret_cast<int4*>(&sm.S[ly * TW + 4 * lane]) = v;
            if (MODE == MODE_SW) {
                const int i = y * L + x;
                const int vv[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
                for (int j = 0; j < 4; ++j)
                    if (vv[j] == i + j || tile_local(p, vv[j], base, tw_eff, th_eff) < 0) anchor |= 1u << (4 * r + j);
            }
        }
    }

    if (MODE == MODE_SW) {
        __syncthreads();                                 // nlist = 0 visible
        // compact the anchors of the whole tile into sm.list (warp scan + one shared atomic per warp)
        const int cnt = __popc(anchor);
        int incl = cnt;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += t;
        }
        int wbase = 0;
        if (lane == 31) wbase = atomicAdd(&sm.nlist, incl);
        wbase = __shfl_sync(0xffffffffu, wbase, 31);
        int pos = wbase + incl - cnt;
        for (uint32_t m = anchor; m; m &= m - 1) {
            const int b = __ffs(m) - 1;
            sm.list[pos++] = (uint16_t)((ly0 + (b >> 2)) * TW + 4 * lane + (b & 3));
        }
        __syncthreads();
        // one Philox draw per anchor, balanced over the CTA
        const int n = sm.nlist;
        for (int k = threadIdx.x; k < n; k += NTHREADS) {
            const int l = sm.list[k];
            sm.st[l] = (uint8_t)flip_state(p, sm.S[l]);
        }
    }
    __syncthreads();

    int nroots = 0, nflip = 0;
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int ly = ly0 + r, y = y0 + ly;
        if (y < L && colv) {
            const int4 v = *reinterpret_cast<const int4*>(&sm.S[ly * TW + 4 * lane]);
            const int vv[4] = {v.x, v.y, v.z, v.w};
            int ww[4];
            uint32_t st[4];
            uint32_t old = 0;
            if (MODE == MODE_WOLFF) old = spins_w[((size_t)y * L + x) >> 2];
            const int i = y * L + x;
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                if (j > 0 && vv[j] == vv[j - 1]) { ww[j] = ww[j - 1]; st[j] = st[j - 1]; }
                else if (MODE == MODE_SW) {
                    int l = ly * TW + 4 * lane + j;      // my own slot if I am an anchor
                    int w = vv[j];
                    if (!((anchor >> (4 * r + j)) & 1u)) {
                        l = tile_local(p, vv[j], base, tw_eff, th_eff);   // >= 0: non-anchors point into the tile
                        w = sm.S[l];
                        const int lw = tile_local(p, w, base, tw_eff, th_eff);
                        if (lw >= 0) l = lw;             // root inside the tile: its own slot; else the hooked local root's
                    }
                    ww[j] = w;
                    st[j] = sm.st[l];
                } else {
                    const int l = tile_local(p, vv[j], base, tw_eff, th_eff);
                    ww[j] = l >= 0 ? sm.S[l] : vv[j];
                    st[j] = 0;
                }
                nroots += (ww[j] == i + j);
            }
            *reinterpret_cast<int4*>(labels + (size_t)y * L + x) = make_int4(ww[0], ww[1], ww[2], ww[3]);
            if (MODE == MODE_SW) {
                uint32_t word = st[0] | (st[1] << 8) | (st[2] << 16) | (st[3] << 24);
                if (p.q == 2) word = 0x01010101u | (word * 0xFEu);   // k=0 -> +1 (0x01), k=1 -> -1 (0xFF)
                spins_w[((size_t)y * L + x) >> 2] = word;
            } else if (MODE == MODE_WOLFF) {
                uint32_t m = 0;                          // bytes to negate
#pragma unroll
                for (int j = 0; j < 4; ++j) if (ww[j] == r0) { m |= 0xFFu << (8 * j); ++nflip; }
                if (m) spins_w[((size_t)y * L + x) >> 2] = __vneg4(old & m) | (old & ~m);
            }
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        nroots += __shfl_xor_sync(0xffffffffu, nroots, o);
        if (MODE == MODE_WOLFF) nflip += __shfl_xor_sync(0xffffffffu, nflip, o);
    }
    if (lane == 0) {
        if (nroots) atomicAdd(&acc->n_clusters, (unsigned long long)nroots);
        if (MODE == MODE_WOLFF && nflip) atomicAdd(wolff_size, (unsigned long long)nflip);
    }
}

}  // namespace swb
