// label_kernels.cuh -- the Swendsen-Wang hot path (S:8a rows a1-a5, a7):
//   k_scan  : bond activation (P:53 step 1, Eq. 7) fused with strip-local labelling: one warp scans a
//             TW x TH strip row by row, the labels of the previous row stay in registers, a run adopts the label of
//             its first contact with the row above, and a (rare) union in a small shared-memory forest happens only
//             when two different trees meet
//   k_seam  : cross-strip consolidation as ONE concurrent union-find pass over the seam bonds
//   k_final : flatten to canonical labels + cluster flip (P:55 step 3) / Wolff flip / label only
// Design notes and the differences from the paper's kernels (self-labelling, hierarchical sewing) are in DESIGN.md.
//
// Provisional label array `prov` (the caller's int32 labels buffer) between k_scan and k_final:
//   entry < 0  : REF | l  -- the site's strip-local ROOT is the site with strip-local index l = ly * TW + lx of the
//                SAME strip, l smaller than the site's own local index (k_scan flattens its forest before it writes)
//   entry >= 0 : global site index g <= own index; g == own index: the site is the root of its tree.  Only
//                strip-local roots carry entries >= 0; k_seam hooks them to roots of other strips (always to a smaller
//                global index), so the root of every tree is the minimum site index of its cluster.
#pragma once
#include "common.cuh"

namespace swb {

constexpr int REF = (int)0x80000000;
constexpr int LMASK = TW * TH - 1;
constexpr int NONE = 0x7FFFFFFF;                         // "no contact" (any value >= 0 works)
constexpr unsigned FULLM = 0xffffffffu;

__device__ __forceinline__ int strip_gidx(int base, int L, int l) { return base + (l >> TW_LOG) * L + (l & (TW - 1)); }

// ------------------------------------------------------------------------------------------------ k_scan
// The strip's forest: one uint16 per strip-local site index.  Entry of a node = its parent node (itself: root); entry
// of any other site = the name (node) it adopted.  Private to one warp.
//
// find with path halving over node entries.  Plain loads/stores, see the 3-phase protocol in unite_batch.
__device__ __forceinline__ int nm_find(volatile uint16_t* nm, int x)
{
    int p = nm[x];
    while (p != x) {
        const int gp = nm[p];
        if (gp == p) return p;
        nm[x] = (uint16_t)gp;
        x = gp;
        p = nm[x];
    }
    return x;
}

// Unite up to 32 queued pairs of names, one per lane (pair = a << 16 | b), hooking the larger root under the smaller.
// 3-phase protocol, no atomics (the forest belongs to this warp): (1) all lanes find roots -- nobody hooks, so a root
// stays a root; (2) hook with a plain store -- lanes hooking the same root collide, one store wins; (3) re-read: losers
// retry from the new roots.
__device__ __forceinline__ void unite_batch(volatile uint16_t* nm, bool have, uint32_t pair)
{
    int ua = (int)(pair >> 16), ub = (int)(pair & 0xFFFFu);
    while (__any_sync(FULLM, have)) {
        if (have) {
            ua = nm_find(nm, ua);
            ub = nm_find(nm, ub);
            if (ua == ub) have = false;
            else if (ua < ub) { const int t = ua; ua = ub; ub = t; }
        }
        __syncwarp();
        if (have) nm[ua] = (uint16_t)ub;
        __syncwarp();
        if (have && nm[ua] == ub) have = false;
    }
}

constexpr int QCAP = 32 + TW;                            // < 32 pairs carried over + at most one new pair per site of a row

// One warp per TW x TH strip, lane -> 4 consecutive columns, rows in sequence.  FROM_BONDS=false: read spins, draw
// bonds (a1).  FROM_BONDS=true: read packed bonds (sw_label).  Writes the flattened strip-local labelling described
// above, the bonds that cross the strip's east / north edge into seamE / seamN (one byte per seam site), and adds the
// number of active bonds to acc->n_active.
//
// Pass 1, row by row.  A "node" is a horizontal run (inside the strip) that has no active north bond from the row
// above; it is named by its first site.  Every other run adopts the name carried by its leftmost contact with the row
// above, so every name is a node.  When a run has further contacts whose names differ from the adopted one, the pair
// of names is queued; queued pairs are united 32 at a time (all lanes busy) in the strip's forest.  Names never depend
// on the forest, so the row loop has no divergent part.
// Pass 2, row by row: every site looks up the root of its name (the rows above are already flat, so this is one load
// unless the name is a node of the same row), the row's entries are overwritten by their roots, and the row is written
// to `prov` as REF | root (or the site's global index if it is the root: hooking is larger-under-smaller, so the root
// is the minimum site index of the strip-local component).
template <bool FROM_BONDS>
__global__ void __launch_bounds__(SCAN_THREADS)
k_scan(const Params p, const uint32_t* __restrict__ spins_w, const uint8_t* __restrict__ bonds_in, int* prov,
       uint8_t* __restrict__ seamE, uint8_t* __restrict__ seamN, Acc* __restrict__ acc)
{
    __shared__ __align__(16) uint16_t s_nm[SCAN_WARPS][TW * TH];
    __shared__ uint32_t s_q[SCAN_WARPS][QCAP];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int tx = blockIdx.x * SCAN_WARPS + warp, ty = blockIdx.y;
    if (tx >= p.ntx) return;                             // no block-wide barrier in this kernel
    uint16_t* nm = s_nm[warp];
    volatile uint16_t* vnm = nm;
    volatile uint32_t* q = s_q[warp];
    const int L = p.L, Lw = L >> 2;
    const int x0 = tx * TW, y0 = ty * TH;
    const int tw_eff = min(TW, L - x0), th_eff = min(TH, L - y0);
    const int x = x0 + 4 * lane;
    const bool colv = 4 * lane < tw_eff;
    const int last_lane = (tw_eff >> 2) - 1;             // lane that owns the strip's last column
    const bool is_last = lane == last_lane;
    const int xw = x >> 2;
    const int xew = ((x + 4 == L) ? 0 : x + 4) >> 2;     // east halo word of the last lane (periodic)
    const unsigned lt = lanemask_lt(), me = 1u << lane, le = lt | me, gt = ~le;

    // spin words of rows y, y+1, y+2 (w*) and the east halo words of the last lane (h*); row index L wraps to 0
    uint32_t w0 = 0, w1 = 0, w2 = 0, h0 = 0, h1 = 0, h2 = 0;
    if (!FROM_BONDS) {
        const int yend = y0 + th_eff;                    // north neighbour row of the strip's last row
        if (colv) {
            w0 = spins_w[(size_t)y0 * Lw + xw];
            if (is_last) h0 = spins_w[(size_t)y0 * Lw + xew];
            const int ya = y0 + 1, yb = y0 + 2;
            if (ya <= yend) { const int yy = ya == L ? 0 : ya; w1 = spins_w[(size_t)yy * Lw + xw]; if (is_last) h1 = spins_w[(size_t)yy * Lw + xew]; }
            if (yb <= yend) { const int yy = yb == L ? 0 : yb; w2 = spins_w[(size_t)yy * Lw + xw]; if (is_last) h2 = spins_w[(size_t)yy * Lw + xew]; }
        }
    }

    int Lp0 = NONE, Lp1 = NONE, Lp2 = NONE, Lp3 = NONE;  // names carried by the previous row's sites
    uint32_t np = 0;                                     // active north bonds from the previous row into this row
    int nact = 0;
    int qn = 0;                                          // queued pairs (warp-uniform)

    for (int ly = 0; ly < th_eff; ++ly) {
        const int y = y0 + ly;
        uint32_t e4 = 0, n4 = 0;
        if (!FROM_BONDS) {
            uint32_t w3 = 0, h3 = 0;                     // prefetch row y+3
            {
                const int yc = y + 3;
                if (colv && yc <= y0 + th_eff) {
                    const int yy = yc == L ? 0 : yc;
                    w3 = spins_w[(size_t)yy * Lw + xw];
                    if (is_last) h3 = spins_w[(size_t)yy * Lw + xew];
                }
            }
            uint32_t wnext = __shfl_down_sync(FULLM, w0, 1);
            if (is_last) wnext = h0;
            if (colv) {
                const uint32_t east = __funnelshift_r(w0, wnext, 8);
                const uint32_t eqe = eq_bytes4(w0, east);
                const uint32_t eqn = eq_bytes4(w0, w1);
                const uint32_t c0 = (uint32_t)(y * L + x) >> 1;
                uint32_t a0, a1, a2, a3, b0, b1, b2, b3;
                philox4x32_10(p, c0, p.t_lo, p.t_hi, DOM_BOND, a0, a1, a2, a3);
                philox4x32_10(p, c0 + 1, p.t_lo, p.t_hi, DOM_BOND, b0, b1, b2, b3);
                const uint32_t de = (a0 < p.T) | ((a2 < p.T) << 1) | ((b0 < p.T) << 2) | ((b2 < p.T) << 3);
                const uint32_t dn = (a1 < p.T) | ((a3 < p.T) << 1) | ((b1 < p.T) << 2) | ((b3 < p.T) << 3);
                e4 = eqe & de;
                n4 = eqn & dn;
                nact += __popc(e4) + __popc(n4);
            }
            w0 = w1; w1 = w2; w2 = w3; h0 = h1; h1 = h2; h2 = h3;
        } else if (colv) {
            const uint32_t b = bonds_in[((size_t)y * L + x) >> 2];
            e4 = (b & 1) | ((b >> 1) & 2) | ((b >> 2) & 4) | ((b >> 3) & 8);
            n4 = ((b >> 1) & 1) | ((b >> 2) & 2) | ((b >> 3) & 4) | ((b >> 4) & 8);
        }

        // bonds that leave the strip go to the seam arrays and are dropped here
        if (colv) {
            if (is_last) {
                seamE[(size_t)tx * L + y] = (uint8_t)(e4 >> 3);
                e4 &= 7u;
            }
            if (ly == th_eff - 1) {
                *reinterpret_cast<uint32_t*>(seamN + (size_t)ty * L + x) = bits_to_bytes4(n4);
                n4 = 0;
            }
        }

        // ---- names of this row's sites ----------------------------------------------------------------------
        const bool E0 = e4 & 1u, E1 = e4 & 2u, E2 = e4 & 4u, E3 = e4 & 8u;
        const bool full = (e4 & 7u) == 7u;
        const bool EL = (__shfl_up_sync(FULLM, e4, 1) & 8u) && lane;
        const int ref0 = REF | (ly * TW + 4 * lane);
        // leftmost contact of every intra-lane segment: forward pass, then spread back from the segment end
        const int c0 = (np & 1u) ? Lp0 : NONE, c1 = (np & 2u) ? Lp1 : NONE;
        const int c2 = (np & 4u) ? Lp2 : NONE, c3 = (np & 8u) ? Lp3 : NONE;
        const int f1 = (E0 && c0 < 0) ? c0 : c1;
        const int f2 = (E1 && f1 < 0) ? f1 : c2;
        const int f3 = (E2 && f2 < 0) ? f2 : c3;
        const int g2 = E2 ? f3 : f2;
        const int g1 = E1 ? g2 : f1;
        const int g0 = E0 ? g1 : c0;
        const int s1 = E0 ? 0 : 1, s2 = E1 ? s1 : 2, s3 = E2 ? s2 : 3;      // first site of each site's segment
        const int pubP = g0;                                                // my prefix segment: contact or NONE
        const int pubS = f3 < 0 ? f3 : ref0 + s3;                           // my suffix segment: contact or new node

        // runs that cross lane boundaries: lanes a..b, a's suffix segment, full lanes, b's prefix segment
        const unsigned LINK = __ballot_sync(FULLM, E3);
        const unsigned FULLB = __ballot_sync(FULLM, full);
        const unsigned CS = __ballot_sync(FULLM, f3 < 0);
        const unsigned CP = __ballot_sync(FULLM, g0 < 0);
        const unsigned nPTL = ~(FULLB & (LINK << 1));                       // lanes where a run cannot pass to the left
        const unsigned nPTR = ~(FULLB & LINK);                              // ... to the right
        const int a_le = 31 - __clz(nPTL & le);                             // bit 0 of nPTL is always set
        const int a_lt = 31 - __clz(nPTL & lt);                             // -1 on lane 0 (unused there: EL = 0)
        const int bS = E3 ? __ffs(nPTR & gt) - 1 : lane;                    // bit 31 of nPTR is always set
        const unsigned MS = (CS & ((1u << bS) - 1u) & (FULLM << a_le)) | (CP & (1u << bS));
        const int srcS = MS ? __ffs(MS) - 1 : a_le;
        const unsigned MP = (CS & lt & (FULLM << (a_lt & 31))) | (CP & me);
        const int srcP = MP ? __ffs(MP) - 1 : a_lt;
        const int vS1 = __shfl_sync(FULLM, pubS, srcS & 31);
        const int vP1 = __shfl_sync(FULLM, pubP, bS);
        const int vS2 = __shfl_sync(FULLM, pubS, srcP & 31);
        const int RS = (srcS == bS) ? vP1 : vS1;                            // name of the run my suffix segment is in
        const int RP = (srcP == lane) ? g0 : vS2;                           // ... my prefix segment (if not full)
        const bool useS = E3 || (full && EL), useP = EL && !full;

        int l0 = g0 < 0 ? g0 : ref0;
        int l1 = g1 < 0 ? g1 : ref0 + s1;
        int l2 = g2 < 0 ? g2 : ref0 + s2;
        int l3 = f3 < 0 ? f3 : ref0 + s3;
        if (useP) { l0 = RP; if (s1 == 0) l1 = RP; if (s2 == 0) l2 = RP; }
        if (useS) { l3 = RS; if (s2 == s3) l2 = RS; if (s1 == s3) l1 = RS; if (s3 == 0) l0 = RS; }

        // the row's entries in the forest: a new node's name is its own index, i.e. it starts as a root
        if (colv) {
            uint2 o;
            o.x = ((uint32_t)l0 & 0xFFFFu) | ((uint32_t)l1 << 16);
            o.y = ((uint32_t)l2 & 0xFFFFu) | ((uint32_t)l3 << 16);
            *reinterpret_cast<uint2*>(nm + ly * TW + 4 * lane) = o;
        }

        // contacts whose carried name differs from the adopted one: queue the pair of names
        unsigned um = ((np & 1u) && Lp0 != l0 ? 1u : 0u) | ((np & 2u) && Lp1 != l1 ? 2u : 0u) |
                      ((np & 4u) && Lp2 != l2 ? 4u : 0u) | ((np & 8u) && Lp3 != l3 ? 8u : 0u);
        unsigned B = __ballot_sync(FULLM, um != 0);
        while (B) {
            if (um) {
                const int c = __ffs(um) - 1;
                um &= um - 1;
                const uint32_t ua = (uint32_t)(c == 0 ? Lp0 : c == 1 ? Lp1 : c == 2 ? Lp2 : Lp3) & 0xFFFFu;
                const uint32_t ub = (uint32_t)(c == 0 ? l0 : c == 1 ? l1 : c == 2 ? l2 : l3) & 0xFFFFu;
                q[qn + __popc(B & lt)] = (ua << 16) | ub;
            }
            qn += __popc(B);
            B = __ballot_sync(FULLM, um != 0);
        }
        if (qn >= 32) {
            __syncwarp();                                // queue and row entries visible to the whole warp
            do {
                qn -= 32;
                unite_batch(vnm, true, q[qn + lane]);
            } while (qn >= 32);
        }

        Lp0 = l0; Lp1 = l1; Lp2 = l2; Lp3 = l3;
        np = n4;
    }

    __syncwarp();
    if (qn > 0) {
        const bool have = lane < qn;
        unite_batch(vnm, have, have ? q[lane] : 0u);
    }
    __syncwarp();

    // ---- pass 2: flatten row by row and write the strip's labels ------------------------------------------------
    for (int ly = 0; ly < th_eff; ++ly) {
        const int lb = ly * TW + 4 * lane;
        const int rowb = ly * TW;
        int r0 = 0, r1 = 0, r2 = 0, r3 = 0;
        if (colv) {
            const uint2 v = *reinterpret_cast<const uint2*>(nm + lb);
            const int n0 = v.x & 0xFFFFu, n1 = v.x >> 16, n2 = v.y & 0xFFFFu, n3 = v.y >> 16;
            // names of the rows above are flat already: one load; a node of this row may be hooked anywhere: chase
            r0 = vnm[n0];
            if (n0 >= rowb) { int t = vnm[r0]; while (t != r0) { r0 = t; t = vnm[r0]; } }
            if (n1 == n0) r1 = r0;
            else { r1 = vnm[n1]; if (n1 >= rowb) { int t = vnm[r1]; while (t != r1) { r1 = t; t = vnm[r1]; } } }
            if (n2 == n1) r2 = r1;
            else { r2 = vnm[n2]; if (n2 >= rowb) { int t = vnm[r2]; while (t != r2) { r2 = t; t = vnm[r2]; } } }
            if (n3 == n2) r3 = r2;
            else { r3 = vnm[n3]; if (n3 >= rowb) { int t = vnm[r3]; while (t != r3) { r3 = t; t = vnm[r3]; } } }
        }
        __syncwarp();                                    // all reads of this row's entries done before they change
        if (colv) {
            uint2 o;
            o.x = (uint32_t)r0 | ((uint32_t)r1 << 16);
            o.y = (uint32_t)r2 | ((uint32_t)r3 << 16);
            *reinterpret_cast<uint2*>(nm + lb) = o;
            const int gi = (y0 + ly) * L + x;
            int4 g;
            g.x = r0 == lb ? gi : (REF | r0);
            g.y = r1 == lb + 1 ? gi + 1 : (REF | r1);
            g.z = r2 == lb + 2 ? gi + 2 : (REF | r2);
            g.w = r3 == lb + 3 ? gi + 3 : (REF | r3);
            *reinterpret_cast<int4*>(prov + (size_t)gi) = g;
        }
        __syncwarp();                                    // the flat entries are visible to the next row
    }

    if (!FROM_BONDS) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) nact += __shfl_xor_sync(FULLM, nact, o);
        if (lane == 0 && nact) atomicAdd(&acc->n_active, (unsigned long long)nact);
    }
}

// ------------------------------------------------------------------------------------------------ seams
// Seam site id -> the two end sites of its crossing bond and the origins of the strips they lie in.
// ids [0, ntx*L): east seams (strip column tc, row y); ids [ntx*L, (ntx+nty)*L): north seams (strip row tr, column x).
__device__ __forceinline__ void seam_sites(const Params& p, int id, int& a, int& b, int& base_a, int& base_b)
{
    const int L = p.L;
    const int nE = p.ntx * L;
    if (id < nE) {
        const int tc = div_L(p, (uint32_t)id), y = id - tc * L;
        const int xs = min((tc + 1) * TW, L) - 1;
        const int xb = xs + 1 == L ? 0 : xs + 1;
        const int yb0 = (y >> TH_LOG) << TH_LOG;
        a = y * L + xs;
        b = y * L + xb;
        base_a = yb0 * L + tc * TW;
        base_b = yb0 * L + xb;
    } else {
        const int k = id - nE;
        const int tr = div_L(p, (uint32_t)k), x = k - tr * L;
        const int ys = min((tr + 1) * TH, L) - 1;
        const int yb = ys + 1 == L ? 0 : ys + 1;
        const int xb0 = (x >> TW_LOG) << TW_LOG;
        a = ys * L + x;
        b = yb * L + x;
        base_a = tr * TH * L + xb0;
        base_b = yb * L + xb0;
    }
}

// strip-local root (global index) of `site`: follow the strip-local references
__device__ __forceinline__ int strip_root(const int* prov, int L, int site, int base)
{
    int cur = site;
    int v = __ldcg(prov + cur);
    while (v < 0) {
        cur = strip_gidx(base, L, v & LMASK);
        v = __ldcg(prov + cur);
    }
    return cur;
}

// Lock-free union by minimum index over the strip-local roots (entries >= 0).  Invariant: entry[x] <= x, and an entry
// only ever changes to a smaller index of the same (growing) set, so a stale read is still an ancestor.  Path halving
// writes an ancestor with a plain store; it can race with the atomicMin of a retrying hook, which then still unites
// the displaced parent.
__device__ __forceinline__ int gfind_halve(int* prov, int x)
{
    int pp = __ldcg(prov + x);
    while (pp != x) {
        const int gp = __ldcg(prov + pp);
        if (gp == pp) return pp;
        prov[x] = gp;
        x = gp;
        pp = __ldcg(prov + x);
    }
    return x;
}

__device__ __forceinline__ int gfind(const int* prov, int x)
{
    int pp = __ldcg(prov + x);
    while (pp != x) { x = pp; pp = __ldcg(prov + x); }
    return x;
}

__device__ __forceinline__ void gunite(int* prov, int a, int b)
{
    while (true) {
        a = gfind_halve(prov, a);
        b = gfind_halve(prov, b);
        if (a == b) return;
        if (a < b) { const int t = a; a = b; b = t; }    // a > b: hook a under b
        const int old = atomicMin(prov + a, b);
        if (old == a) return;                            // a was a root and now points to b
        a = old;                                         // a had been hooked meanwhile: entry = min(old,b); join old and b
    }
}

// One thread per seam site: if its crossing bond is active, unite the strip-local roots of its two ends.
// `seam` is seamE followed by seamN (contiguous).
__global__ void __launch_bounds__(256)
k_seam(const Params p, const uint8_t* __restrict__ seam, int* prov)
{
    const int nseam = (p.ntx + p.nty) * p.L;
    const int id = blockIdx.x * blockDim.x + threadIdx.x;
    const bool on = id < nseam && seam[id];
    int ra = -1, rb = -1;
    if (on) {
        int a, b, base_a, base_b;
        seam_sites(p, id, a, b, base_a, base_b);
        ra = strip_root(prov, p.L, a, base_a);
        rb = strip_root(prov, p.L, b, base_b);
    }
    // the previous seam site joins the same two strip-local clusters: skip (its thread does the union)
    const int pa = __shfl_up_sync(FULLM, ra, 1), pb = __shfl_up_sync(FULLM, rb, 1);
    const bool dup = (threadIdx.x & 31) != 0 && pa == ra && pb == rb;
    if (on && !dup) gunite(prov, ra, rb);
}

// ------------------------------------------------------------------------------------------------ k_final
enum { MODE_SW = 0, MODE_WOLFF = 1, MODE_LABEL = 2 };

__device__ __forceinline__ uint32_t flip_state(const Params& p, int root)
{
    uint32_t w0, w1, w2, w3;
    philox4x32_10(p, (uint32_t)root, p.t_lo, p.t_hi, DOM_FLIP, w0, w1, w2, w3);
    return __umulhi(w0, (uint32_t)p.q);                  // uniform state in [0,q)  (S:8c.6)
}

// Shared memory of k_final: the strip's forest, one state byte per strip-local root, the compacted list of roots.
struct FinalSmem {
    int      S[TW * TH];
    uint16_t list[TW * TH];
    uint8_t  st[TW * TH];
    int      nlist;
    int      r0;
};

// One CTA per strip: canonical labels (root of every site) + the new spins.
//   MODE_SW    : s_i = state drawn for the root (assign, P:55 step 3)
//   MODE_WOLFF : s_i = -s_i iff root(i) == root(seed site i0); adds |C| to *wolff_size
//   MODE_LABEL : labels only
// Strip-local roots (entries >= 0) are compacted into a list; each is resolved to the root of its global tree (a
// chase over entries >= 0 of other strips, which concurrently running CTAs may already have overwritten with final
// labels -- those are roots of the same tree, so the chase still ends at the right root) and draws one Philox state.
// Every other site follows its strip-local references through shared memory.
template <int MODE>
__global__ void __launch_bounds__(FIN_THREADS)
k_final(const Params p, int* labels, uint32_t* __restrict__ spins_w, Acc* __restrict__ acc,
        unsigned long long* __restrict__ wolff_size)
{
    __shared__ __align__(16) FinalSmem sm;
    constexpr int R = TH / FIN_WARPS;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int L = p.L;
    const int x0 = blockIdx.x * TW, y0 = blockIdx.y * TH;
    const int tw_eff = min(TW, L - x0);
    const int x = x0 + 4 * lane;
    const bool colv = 4 * lane < tw_eff;
    const int ly0 = warp * R;
    const int base = y0 * L + x0;

    if (threadIdx.x == 0) {
        sm.nlist = 0;
        if (MODE == MODE_WOLFF) {
            uint32_t w0, w1, w2, w3;
            philox4x32_10(p, 0u, p.t_lo, p.t_hi, DOM_WSEED, w0, w1, w2, w3);
            const int i0 = (int)__umulhi(w0, (uint32_t)p.N);
            const int iy = i0 / L, ix = i0 - iy * L;
            const int b0 = ((iy >> TH_LOG) << TH_LOG) * L + ((ix >> TW_LOG) << TW_LOG);
            sm.r0 = gfind(labels, strip_root(labels, L, i0, b0));
        }
    }

    uint32_t rootm = 0;                                  // bit 4r+j: my site (row r, column j) is a strip-local root
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int ly = ly0 + r, y = y0 + ly;
        if (y < L && colv) {
            const int4 v = *reinterpret_cast<const int4*>(labels + (size_t)y * L + x);
            *reinterpret_cast<int4*>(&sm.S[ly * TW + 4 * lane]) = v;
            const int i = y * L + x;
            if (MODE == MODE_SW)
                rootm |= ((v.x >= 0) | ((v.y >= 0) << 1) | ((v.z >= 0) << 2) | ((v.w >= 0) << 3)) << (4 * r);
            else                                         // only hooked roots need work
                rootm |= ((v.x >= 0 && v.x != i) | ((v.y >= 0 && v.y != i + 1) << 1) | ((v.z >= 0 && v.z != i + 2) << 2) |
                          ((v.w >= 0 && v.w != i + 3) << 3)) << (4 * r);
        }
    }
    __syncthreads();                                     // nlist = 0, r0 and S visible

    // compact the roots of the whole strip into sm.list (warp scan + one shared atomic per warp)
    {
        const int cnt = __popc(rootm);
        int incl = cnt;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(FULLM, incl, o);
            if (lane >= o) incl += t;
        }
        int wbase = 0;
        if (lane == 31 && incl) wbase = atomicAdd(&sm.nlist, incl);
        wbase = __shfl_sync(FULLM, wbase, 31);
        int pos = wbase + incl - cnt;
        for (uint32_t m = rootm; m; m &= m - 1) {
            const int b = __ffs(m) - 1;
            sm.list[pos++] = (uint16_t)((ly0 + (b >> 2)) * TW + 4 * lane + (b & 3));
        }
    }
    __syncthreads();
    // one global resolve + one Philox draw per strip-local root, balanced over the CTA
    {
        const int n = sm.nlist;
        for (int k = threadIdx.x; k < n; k += FIN_THREADS) {
            const int l = sm.list[k];
            int v = sm.S[l];
            if (v != strip_gidx(base, L, l)) {           // hooked by k_seam: find the root of the global tree
                v = gfind(labels, v);
                sm.S[l] = v;
            }
            if (MODE == MODE_SW) sm.st[l] = (uint8_t)flip_state(p, v);
        }
    }
    __syncthreads();

    const int r0 = MODE == MODE_WOLFF ? sm.r0 : -1;
    int nroots = 0, nflip = 0;
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int ly = ly0 + r, y = y0 + ly;
        if (y < L && colv) {
            const int lb = ly * TW + 4 * lane;
            const int4 v = *reinterpret_cast<const int4*>(&sm.S[lb]);
            const int vv[4] = {v.x, v.y, v.z, v.w};
            int ww[4];
            uint32_t st[4];
            uint32_t old = 0;
            if (MODE == MODE_WOLFF) old = spins_w[((size_t)y * L + x) >> 2];
            const int i = y * L + x;
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                if (j > 0 && vv[j] == vv[j - 1] && vv[j] < 0) { ww[j] = ww[j - 1]; st[j] = st[j - 1]; }
                else {
                    int l = lb + j, w = vv[j];
                    if (w < 0) { l = w & LMASK; w = sm.S[l]; }     // k_scan wrote flat references: one hop
                    ww[j] = w;
                    st[j] = MODE == MODE_SW ? sm.st[l] : 0u;
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
        nroots += __shfl_xor_sync(FULLM, nroots, o);
        if (MODE == MODE_WOLFF) nflip += __shfl_xor_sync(FULLM, nflip, o);
    }
    if (lane == 0) {
        if (nroots) atomicAdd(&acc->n_clusters, (unsigned long long)nroots);
        if (MODE == MODE_WOLFF && nflip) atomicAdd(wolff_size, (unsigned long long)nflip);
    }
}

}  // namespace swb
