// label_kernels.cuh -- the Swendsen-Wang hot path (S:8a rows a1-a5, a7):
//   k_scan  : bond activation (P:53 step 1, Eq. 7) fused with strip-local labelling: one warp scans a
//             TW x TH strip row by row, the names of the previous row stay in registers, a run adopts the name of its
//             first contact with the row above; pairs of names that meet are queued and united 32 at a time in a small
//             shared-memory forest.  The roots of the strip's edge sites go to compact edge arrays.
//   k_seam  : cross-strip consolidation as ONE concurrent union-find pass over the seam bonds
//   k_final : flatten to canonical labels + cluster flip (P:55 step 3) / Wolff flip / label only
// Design notes and the differences from the paper's kernels (self-labelling, hierarchical sewing) are in DESIGN.md.
//
// Provisional label array `prov` (the caller's int32 labels buffer) between k_scan and k_final.  A "node" is a site
// that names a run (see k_scan); every strip-local tree is a tree of nodes.
//   entry >= 0            : the site is a node and the root of its strip-local tree; the value is a global site index
//                           g <= own index (g == own index: root of its global tree; k_seam hooks roots of different
//                           strips, always under a smaller global index, so the root of every tree is the minimum site
//                           index of its cluster)
//   entry = REF|HOOK|l    : the site is a node that was hooked under the node with strip-local index l < own
//   entry = REF|l         : the site is not a node; it belongs to the tree of the node with strip-local index l
// with l = ly * TW + lx inside the SAME strip.
#pragma once
#include "common.cuh"

namespace swb {

constexpr int REF = (int)0x80000000;
constexpr int HOOK = 0x40000000;
constexpr int LMASK = TW * TH - 1;
constexpr int NONE = 0x7FFFFFFF;                         // "no contact" (any value >= 0 works)
constexpr unsigned FULLM = 0xffffffffu;

__device__ __forceinline__ int strip_gidx(int base, int L, int l) { return base + (l >> TW_LOG) * L + (l & (TW - 1)); }

// ------------------------------------------------------------------------------------------------ k_scan
// The strip's forest: one uint16 per strip-local site index.  Entry of a node = its parent node (itself: root); entry
// of any other site = the name (node) it adopted, so a chase that starts at any site ends at the root of its tree.
// Private to one warp.
//
// find with path halving.  Plain loads/stores: halving rewrites non-root entries with an ancestor (concurrent lanes may
// interleave, every value written is an ancestor); roots change only in phase 2 of unite_batch.
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

// roots of four sites in lockstep (four independent chases per iteration)
__device__ __forceinline__ void nm_root4(const volatile uint16_t* nm, int& a, int& b, int& c, int& d)
{
    int pa = nm[a], pb = nm[b], pc = nm[c], pd = nm[d];
    while ((pa ^ a) | (pb ^ b) | (pc ^ c) | (pd ^ d)) {
        a = pa; b = pb; c = pc; d = pd;
        pa = nm[a]; pb = nm[b]; pc = nm[c]; pd = nm[d];
    }
}

// Unite one queued pair of names per lane (pair = a << 16 | b), hooking the larger root under the smaller and writing
// every hook through to `prov`.  3-phase protocol, no atomics (the forest belongs to this warp): (1) all lanes find
// roots -- nobody hooks, so a root stays a root; (2) hook with a plain store -- lanes hooking the same root collide, one
// store wins; (3) re-read: losers retry from the new roots.
__device__ __forceinline__ void unite_batch(volatile uint16_t* nm, bool have, uint32_t pair, int* prov, int base, int L)
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
        if (have && nm[ua] == ub) {
            prov[strip_gidx(base, L, ua)] = REF | HOOK | ub;
            have = false;
        }
    }
}

constexpr int QCAP = 32 + TW;                            // < 32 pairs carried over + at most one new pair per site of a row

// Edge arrays (workspace): for every site on the edge of a strip the global index of its strip-local root.
//   edgeA = [ rootE (ntx * L) | rootN (nty * L) ] : last column of strip column tc at row y -> [tc * L + y], last row of
//           strip row tr at column x -> [ntx * L + tr * L + x]; the value is -1 if the bond that leaves the strip there
//           (east bond of the last column, north bond of the last row) is not active
//   edgeB = [ rootW (ntx * L) | rootS (nty * L) ] : first column / first row, same indexing
//
// One warp per TW x TH strip, lane -> 4 consecutive columns, rows in sequence.  FROM_BONDS=false: read spins, draw
// bonds (a1).  FROM_BONDS=true: read packed bonds (sw_label).  Writes the provisional labels described above and the
// edge arrays, and adds the number of active bonds to acc->n_active.
//
// Row step.  A "node" is a horizontal run (inside the strip) that has no active north bond from the row above; it is
// named by its first site.  Every other run adopts the name carried by its leftmost contact with the row above, so
// every name is a node.  When a run has further contacts whose names differ from the adopted one, the pair of names is
// queued; queued pairs are united 32 at a time (all lanes busy) in the strip's forest.  Names never depend on the
// forest, so the row loop has no divergent part.
template <bool FROM_BONDS>
__global__ void __launch_bounds__(SCAN_THREADS)
k_scan(const Params p, const uint32_t* __restrict__ spins_w, const uint8_t* __restrict__ bonds_in, int* prov,
       int* __restrict__ edgeA, int* __restrict__ edgeB, Acc* __restrict__ acc)
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
    const int base = y0 * L + x0;
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
    uint32_t eastm = 0;                                  // last lane: bit ly = the east bond that leaves the strip in row ly
    uint32_t northm = 0;                                 // the 4 north bonds that leave the strip in the last row

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

        // bonds that leave the strip are remembered for the edge arrays and dropped here
        if (is_last) {
            eastm |= (e4 >> 3) << ly;
            e4 &= 7u;
        }
        if (ly == th_eff - 1) {
            northm = n4;
            n4 = 0;
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

        // the row's entries in the forest (a new node's name is its own index, i.e. it starts as a root) and in `prov`
        if (colv) {
            uint2 o;
            o.x = ((uint32_t)l0 & 0xFFFFu) | ((uint32_t)l1 << 16);
            o.y = ((uint32_t)l2 & 0xFFFFu) | ((uint32_t)l3 << 16);
            *reinterpret_cast<uint2*>(nm + ly * TW + 4 * lane) = o;
            const int gi = y * L + x;
            int4 g;
            g.x = l0 == ref0 ? gi : l0;
            g.y = l1 == ref0 + 1 ? gi + 1 : l1;
            g.z = l2 == ref0 + 2 ? gi + 2 : l2;
            g.w = l3 == ref0 + 3 ? gi + 3 : l3;
            *reinterpret_cast<int4*>(prov + (size_t)gi) = g;
        }

        // contacts whose carried name differs from the adopted one: queue the pair of names
        {
            const bool m0 = (np & 1u) && Lp0 != l0, m1 = (np & 2u) && Lp1 != l1;
            const bool m2 = (np & 4u) && Lp2 != l2, m3 = (np & 8u) && Lp3 != l3;
            const unsigned B0 = __ballot_sync(FULLM, m0), B1 = __ballot_sync(FULLM, m1);
            const unsigned B2 = __ballot_sync(FULLM, m2), B3 = __ballot_sync(FULLM, m3);
            if (m0) q[qn + __popc(B0 & lt)] = __byte_perm((uint32_t)l0, (uint32_t)Lp0, 0x5410);
            qn += __popc(B0);
            if (m1) q[qn + __popc(B1 & lt)] = __byte_perm((uint32_t)l1, (uint32_t)Lp1, 0x5410);
            qn += __popc(B1);
            if (m2) q[qn + __popc(B2 & lt)] = __byte_perm((uint32_t)l2, (uint32_t)Lp2, 0x5410);
            qn += __popc(B2);
            if (m3) q[qn + __popc(B3 & lt)] = __byte_perm((uint32_t)l3, (uint32_t)Lp3, 0x5410);
            qn += __popc(B3);
        }
        if (qn >= 32) {
            __syncwarp();                                // queue, forest entries and `prov` rows visible to the whole warp
            do {
                qn -= 32;
                unite_batch(vnm, true, q[qn + lane], prov, base, L);
            } while (qn >= 32);
            __syncwarp();                                // queue slots read before the next row overwrites them
        }

        Lp0 = l0; Lp1 = l1; Lp2 = l2; Lp3 = l3;
        np = n4;
    }

    __syncwarp();
    if (qn > 0) {
        const bool have = lane < qn;
        unite_batch(vnm, have, have ? q[lane] : 0u, prov, base, L);
    }
    __syncwarp();

    // ---- edge arrays: strip-local roots of the sites on the four edges ----------------------------------------------
    {
        const int nE = p.ntx * L;
        if (colv) {
            // first row -> rootS, last row -> rootN (-1 where the north bond that leaves the strip is not active)
            const int lb0 = 4 * lane, lb1 = (th_eff - 1) * TW + 4 * lane;
            int s0 = lb0, s1 = lb0 + 1, s2 = lb0 + 2, s3 = lb0 + 3;
            int n0 = lb1, n1 = lb1 + 1, n2 = lb1 + 2, n3 = lb1 + 3;
            nm_root4(vnm, s0, s1, s2, s3);
            nm_root4(vnm, n0, n1, n2, n3);
            int4 s, n;
            s.x = strip_gidx(base, L, s0);
            s.y = strip_gidx(base, L, s1);
            s.z = strip_gidx(base, L, s2);
            s.w = strip_gidx(base, L, s3);
            n.x = (northm & 1u) ? strip_gidx(base, L, n0) : -1;
            n.y = (northm & 2u) ? strip_gidx(base, L, n1) : -1;
            n.z = (northm & 4u) ? strip_gidx(base, L, n2) : -1;
            n.w = (northm & 8u) ? strip_gidx(base, L, n3) : -1;
            *reinterpret_cast<int4*>(edgeB + (size_t)nE + (size_t)ty * L + x) = s;
            *reinterpret_cast<int4*>(edgeA + (size_t)nE + (size_t)ty * L + x) = n;
        }
        // first column -> rootW, last column -> rootE: lane i takes row i
        const uint32_t em = __shfl_sync(FULLM, eastm, last_lane);
        if (lane < th_eff) {
            int w = lane * TW, e = lane * TW + tw_eff - 1, w2 = w, e2 = e;
            nm_root4(vnm, w, e, w2, e2);
            edgeB[(size_t)tx * L + y0 + lane] = strip_gidx(base, L, w);
            edgeA[(size_t)tx * L + y0 + lane] = ((em >> lane) & 1u) ? strip_gidx(base, L, e) : -1;
        }
    }

    if (!FROM_BONDS) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) nact += __shfl_xor_sync(FULLM, nact, o);
        if (lane == 0 && nact) atomicAdd(&acc->n_active, (unsigned long long)nact);
    }
}

// ------------------------------------------------------------------------------------------------ seams
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
__device__ __forceinline__ int gfind(const int* prov, int x)
{
    int pp = __ldcg(prov + x);
    while (pp != x) { x = pp; pp = __ldcg(prov + x); }
    return x;
}

// Unite the trees of a and b.  Both finds advance in lockstep (two independent loads per round trip), with path halving:
// one round trip when both are roots already, two when each is one hop from its root.
__device__ __forceinline__ void gunite(int* prov, int a, int b)
{
    while (true) {
        while (true) {
            const int pa = __ldcg(prov + a), pb = __ldcg(prov + b);
            if (pa == a && pb == b) break;
            const int ga = __ldcg(prov + pa), gb = __ldcg(prov + pb);
            if (pa != a && ga != pa) prov[a] = ga;       // path halving
            if (pb != b && gb != pb) prov[b] = gb;
            const bool done = ga == pa && gb == pb;      // both parents are roots
            a = ga; b = gb;
            if (done) break;
        }
        if (a == b) return;
        if (a < b) { const int t = a; a = b; b = t; }    // a > b: hook a under b
        const int old = atomicMin(prov + a, b);
        if (old == a) return;                            // a was a root and now points to b
        a = old;                                         // a had been hooked meanwhile: entry = min(old,b); join old and b
    }
}

// One thread per seam site (ids [0, ntx*L): east seams (strip column tc, row y); then nty*L north seams (strip row tr,
// column x)): if its crossing bond is active (edgeA >= 0), unite the strip-local roots of its two ends.  Both edge
// entries are loaded up front (the index of the facing entry does not depend on the first load).
__global__ void __launch_bounds__(256)
k_seam(const Params p, const int* __restrict__ edgeA, const int* __restrict__ edgeB, int* prov)
{
    const int L = p.L;
    const int nE = p.ntx * L, nseam = (p.ntx + p.nty) * L;
    const int id = blockIdx.x * blockDim.x + threadIdx.x;
    int ra = -1, rb = -1;
    if (id < nseam) {
        int idb;
        if (id < nE) {                                   // first column of the strip column to the east (periodic)
            const int tc = div_L(p, (uint32_t)id);
            idb = tc + 1 == p.ntx ? id - tc * L : id + L;
        } else {                                         // first row of the strip row to the north (periodic)
            const int tr = div_L(p, (uint32_t)(id - nE));
            idb = tr + 1 == p.nty ? id - tr * L : id + L;
        }
        ra = edgeA[id];
        rb = edgeB[idb];
    }
    // the previous ACTIVE seam site of this warp joins the same two strip-local clusters: skip (its thread does the union)
    const unsigned act = __ballot_sync(FULLM, ra >= 0);
    const int prev = 31 - __clz(act & lanemask_lt());    // -1: none
    const int pa = __shfl_sync(FULLM, ra, prev & 31), pb = __shfl_sync(FULLM, rb, prev & 31);
    const bool dup = prev >= 0 && pa == ra && pb == rb;
    if (ra >= 0 && !dup) gunite(prov, ra, rb);
}

// ------------------------------------------------------------------------------------------------ k_final
enum { MODE_SW = 0, MODE_WOLFF = 1, MODE_LABEL = 2 };

__device__ __forceinline__ uint32_t flip_state(const Params& p, int root)
{
    uint32_t w0, w1, w2, w3;
    philox4x32_10(p, (uint32_t)root, p.t_lo, p.t_hi, DOM_FLIP, w0, w1, w2, w3);
    return __umulhi(w0, (uint32_t)p.q);                  // uniform state in [0,q)  (S:8c.6)
}

// Shared memory of k_final: the strip's entries (node entries are rewritten in place with the FINAL value of their
// cluster: the canonical label and, in MODE_SW, the cluster's new state above bit Params::sbit -- a value >= 0) and the
// compacted list of the strip-local roots.
struct FinalSmem {
    int      S[TW * TH];
    uint16_t list[TW * TH];
    int      nroot;
    int      r0;
};

// One CTA per strip: canonical labels (root of every site) + the new spins.
//   MODE_SW    : s_i = state drawn for the root (assign, P:55 step 3)
//   MODE_WOLFF : s_i = -s_i iff root(i) == root(seed site i0); adds |C| to *wolff_size
//   MODE_LABEL : labels only
// (1) the strip's entries go to shared memory; the strip-local roots are compacted into a list.  (2) every strip-local
// root is resolved to the root of its global tree (a chase over entries >= 0 of other strips, which concurrently running
// CTAs may already have overwritten with final labels -- those are roots of the same tree, so the chase still ends at the
// right root) and draws one Philox state; its entry becomes the final value.  (3) every hooked node (each thread looks
// after its own sites) follows its references to the first entry >= 0 -- the strip-local root or a hooked node that is
// final already, both carry the final value of the cluster -- and takes that value.  (4) every other site is one hop
// from a node.
template <int MODE>
__global__ void __launch_bounds__(FIN_THREADS, 2048 / FIN_THREADS)
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
    volatile int* S = sm.S;

    if (threadIdx.x == 0) {
        sm.nroot = 0;
        if (MODE == MODE_WOLFF) {
            uint32_t w0, w1, w2, w3;
            philox4x32_10(p, 0u, p.t_lo, p.t_hi, DOM_WSEED, w0, w1, w2, w3);
            const int i0 = (int)__umulhi(w0, (uint32_t)p.N);
            const int iy = i0 / L, ix = i0 - iy * L;
            const int b0 = ((iy >> TH_LOG) << TH_LOG) * L + ((ix >> TW_LOG) << TW_LOG);
            sm.r0 = gfind(labels, strip_root(labels, L, i0, b0));
        }
    }
    __syncthreads();                                     // counter (and r0) visible

    // (1) entries -> shared memory; compact the roots into sm.list
    uint32_t hookm = 0;                                  // bit 4r+j: my site (row r, column j) is a hooked node
    {
        uint32_t rootm = 0;                              // ... is a strip-local root
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int ly = ly0 + r, y = y0 + ly;
            if (y < L && colv) {
                const int4 v = *reinterpret_cast<const int4*>(labels + (size_t)y * L + x);
                *reinterpret_cast<int4*>(&sm.S[ly * TW + 4 * lane]) = v;
                // top bytes of the 4 entries; bit 7 clear: root, bits 7 and 6 set: hooked node; 4 spread bits -> 4 adjacent
                const uint32_t t = __byte_perm(__byte_perm(v.x, v.y, 0x0073), __byte_perm(v.z, v.w, 0x0073), 0x5410);
                rootm |= (((~t & 0x80808080u) * 0x00204081u) >> 28) << (4 * r);
                hookm |= (((t & (t << 1) & 0x80808080u) * 0x00204081u) >> 28) << (4 * r);
            }
        }
        const int cnt = __popc(rootm);
        int incl = cnt;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(FULLM, incl, o);
            if (lane >= o) incl += t;
        }
        int rbase = 0;
        if (lane == 31 && incl) rbase = atomicAdd(&sm.nroot, incl);
        rbase = __shfl_sync(FULLM, rbase, 31);
        int pos = rbase + incl - cnt;
        for (uint32_t m = rootm; m; m &= m - 1) {
            const int b = __ffs(m) - 1;
            sm.list[pos++] = (uint16_t)((ly0 + (b >> 2)) * TW + 4 * lane + (b & 3));
        }
    }
    __syncthreads();
    // (2) one global resolve + one Philox draw per strip-local root, balanced over the CTA
    int nroots = 0;
    {
        const int n = sm.nroot;
        for (int k = threadIdx.x; k < n; k += FIN_THREADS) {
            const int l = sm.list[k];
            int v = sm.S[l];
            const int g = strip_gidx(base, L, l);
            if (v != g) v = gfind(labels, v);            // hooked by k_seam: find the root of the global tree
            nroots += (v == g);
            // final label and, above bit p.sbit, the new state of the cluster (labels are < 2^sbit)
            sm.S[l] = MODE == MODE_SW ? (int)((uint32_t)v | (flip_state(p, v) << p.sbit)) : v;
        }
    }
    __syncthreads();
    // (3) my hooked nodes
    for (uint32_t m = hookm; m; m &= m - 1) {
        const int b = __ffs(m) - 1;
        const int l = (ly0 + (b >> 2)) * TW + 4 * lane + (b & 3);
        int e = S[l];
        do { e = S[e & LMASK]; } while (e < 0);
        S[l] = e;
    }
    __syncthreads();

    // (4) every site
    const int r0 = MODE == MODE_WOLFF ? sm.r0 : -1;
    const int lmask = (1 << p.sbit) - 1;
    int nflip = 0;
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int ly = ly0 + r, y = y0 + ly;
        if (y < L && colv) {
            const int4 v = *reinterpret_cast<const int4*>(&sm.S[ly * TW + 4 * lane]);
            int ww[4] = {v.x, v.y, v.z, v.w};
            uint32_t st[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                int w = ww[j];
                if (w < 0) w = sm.S[w & LMASK];          // not a node: one hop to its node, which is final
                ww[j] = MODE == MODE_SW ? (w & lmask) : w;
                st[j] = MODE == MODE_SW ? (uint32_t)w >> p.sbit : 0u;
            }
            *reinterpret_cast<int4*>(labels + (size_t)y * L + x) = make_int4(ww[0], ww[1], ww[2], ww[3]);
            if (MODE == MODE_SW) {
                uint32_t word = st[0] | (st[1] << 8) | (st[2] << 16) | (st[3] << 24);
                if (p.q == 2) word = 0x01010101u | (word * 0xFEu);   // k=0 -> +1 (0x01), k=1 -> -1 (0xFF)
                spins_w[((size_t)y * L + x) >> 2] = word;
            } else if (MODE == MODE_WOLFF) {
                const uint32_t m = (ww[0] == r0 ? 0xFFu : 0u) | (ww[1] == r0 ? 0xFF00u : 0u) |
                                   (ww[2] == r0 ? 0xFF0000u : 0u) | (ww[3] == r0 ? 0xFF000000u : 0u);   // bytes to negate
                if (m) {
                    const uint32_t old = spins_w[((size_t)y * L + x) >> 2];
                    spins_w[((size_t)y * L + x) >> 2] = __vneg4(old & m) | (old & ~m);
                    nflip += __popc(m) >> 3;
                }
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
