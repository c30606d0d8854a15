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
// Programmatic dependent launch (SWB_PDL 1: k_seam and, in a sweep, k_final; 2: also k_scan, the per-sweep counters being
// zeroed by a one-CTA kernel instead of a memset, so that a chain of sweeps is kernel -> kernel throughout): the kernels are
// launched with programmatic stream serialisation and wait for the preceding kernel's memory at
// cudaGridDependencySynchronize(), so their launch is staged while that kernel still runs.  Measured, us per sweep (0 / 1 / 2):
// L=16384: 1562 / 1557 / 1554; L=4096: 141 / 137 / 134; L=1024: 55.0 / 51.2 / 48.0; L=64: 40.7 / 37.9 / 33.4.  An early
// cudaTriggerProgrammaticLaunchCompletion() in the preceding kernel lets waiting CTAs take slots from it (1596 at L=16384).
#ifndef SWB_PDL
#define SWB_PDL 2
#endif

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
// interleave, every value written is an ancestor); roots change only in phase 2 of unite_batch (scan_kernel.cuh).
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

// Edge arrays (workspace): for every site on the edge of a strip the global index of its strip-local root.
//   edgeA = [ rootE (ntx * L) | rootN (nty * L) ] : last column of strip column tc at row y -> [tc * L + y], last row of
//           strip row tr at column x -> [ntx * L + tr * L + x]; the value is -1 if the bond that leaves the strip there
//           (east bond of the last column, north bond of the last row) is not active
//   edgeB = [ rootW (ntx * L) | rootS (nty * L) ] : first column / first row, same indexing
//
}  // namespace swb

#include "scan_kernel.cuh"

namespace swb {

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

// The same chase in k_final, through the L1 cache: no entry is hooked any more (k_seam has finished; L1 is invalidated at
// the kernel boundary), the only concurrent writes are final labels -- roots of the same tree -- so a stale line is still
// an ancestor.  The root entries of the large clusters are read by every strip they pass through: cached per SM they stop
// being a hot spot in one L2 slice.
__device__ __forceinline__ int gfind_cached(const int* prov, int x)
{
    int pp = __ldca(prov + x);
    while (pp != x) { x = pp; pp = __ldca(prov + x); }
    return x;
}

// Unite the trees of a and b; pa, pb = entries of a and b, loaded by the caller.  Both finds advance in lockstep (two
// independent loads per round trip), with path halving: nothing more to load when both are roots already, one round
// trip when each is one hop from its root.
__device__ __forceinline__ void gunite(int* prov, int a, int b, int pa, int pb)
{
    while (true) {
        while (pa != a || pb != b) {
            const int ga = __ldcg(prov + pa), gb = __ldcg(prov + pb);
            if (pa != a && ga != pa) prov[a] = ga;       // path halving
            if (pb != b && gb != pb) prov[b] = gb;
            const bool done = ga == pa && gb == pb;      // both parents are roots
            a = ga; b = gb;
            if (done) break;
            pa = __ldcg(prov + a); pb = __ldcg(prov + b);
        }
        if (a == b) return;
        if (a < b) { const int t = a; a = b; b = t; }    // a > b: hook a under b
        const int old = atomicMin(prov + a, b);
        if (old == a) return;                            // a was a root and now points to b
        a = old;                                         // a had been hooked meanwhile: entry = min(old,b); join old and b
        pa = __ldcg(prov + a); pb = __ldcg(prov + b);
    }
}

// Seam site `id` (ids [0, ntx*L): east seams (strip column tc, row y); then nty*L north seams (strip row tr, column x)):
// the strip-local roots of its two ends, ra = -1 if its crossing bond is not active.
__device__ __forceinline__ void seam_ends(const Params& p, const int* __restrict__ edgeA, const int* __restrict__ edgeB,
                                          int id, int nE, int nseam, int& ra, int& rb)
{
    ra = -1; rb = -1;
    if (id < nseam) {
        const int L = p.L;
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
}

// true if this lane has a union to do: its bond is active and the previous ACTIVE seam site of the warp does not join the
// same two strip-local clusters (then that lane does the union)
__device__ __forceinline__ bool seam_todo(int ra, int rb)
{
    const unsigned act = __ballot_sync(FULLM, ra >= 0);
    const int prev = 31 - __clz(act & lanemask_lt());    // -1: none
    const int pa = __shfl_sync(FULLM, ra, prev & 31), pb = __shfl_sync(FULLM, rb, prev & 31);
    return ra >= 0 && !(prev >= 0 && pa == ra && pb == rb);
}

// SEAM_PER_THREAD seam sites per thread (id, id + part, ...): all edge entries are loaded up front, then all root
// entries, so that a thread has many independent loads in flight (the kernel is bound by memory latency); then the unions.
#ifndef SWB_SEAM_PER_THREAD
#define SWB_SEAM_PER_THREAD 4
#endif
constexpr int SEAM_PER_THREAD = SWB_SEAM_PER_THREAD;
__host__ __device__ inline int seam_part(int nseam)     // ids per part, a multiple of 32: a warp's ids stay consecutive
{
    return ((nseam + 32 * SEAM_PER_THREAD - 1) / (32 * SEAM_PER_THREAD)) * 32;
}

__host__ __device__ inline int seam_band_sites(const Params& p) { return p.ntx * p.nband * TH + (p.nband - 1) * p.L; }

// series != NULL (a sweep): one thread also files the (sat, minus) totals k_scan has just accumulated under the sweep's
// counter, so that a chain keeps the energy and magnetisation of every configuration it passes through (sw_series_read).
// BAND (multi-GPU row bands, band_kernels.cuh): only the seams INSIDE the band [ty0, ty0 + nband) of strip rows -- east seams of
// its rows, north seams between its strip rows; the north seam on top of the band crosses to another rank.
template <bool BAND>
__global__ void __launch_bounds__(256)
k_seam(const Params p, const int* __restrict__ edgeA, const int* __restrict__ edgeB, int* prov,
       const Acc* __restrict__ acc, SeriesEntry* __restrict__ series)
{
#if SWB_PDL
    cudaGridDependencySynchronize();
#endif
    if (series != nullptr && blockIdx.x == 0 && threadIdx.x == 0) {
        unsigned long long sat = 0, minus = 0;
        for (int k = 0; k < ACC_PARTS; ++k) { sat += acc->part[k].sat; minus += acc->part[k].minus; }
        SeriesEntry e; e.sat = sat; e.minus = minus;
        series[p.t_lo & (SERIES_RING - 1)] = e;
    }
    const int nE = p.ntx * p.L, nseam = (p.ntx + p.nty) * p.L;
    // BAND: threads are enumerated over the band's own seam sites: ntx x (rows of the band) east sites, then the north sites
    // of its strip rows but the last
    const int bh = p.nband * TH, nlocal = BAND ? seam_band_sites(p) : nseam;
    const int part = seam_part(nlocal);
    const int id = blockIdx.x * blockDim.x + threadIdx.x;
    int ra[SEAM_PER_THREAD], rb[SEAM_PER_THREAD], pa[SEAM_PER_THREAD], pb[SEAM_PER_THREAD];
    bool todo[SEAM_PER_THREAD];
#pragma unroll
    for (int k = 0; k < SEAM_PER_THREAD; ++k) {
        int sid = id < part ? id + k * part : nlocal;
        if (BAND) {
            if (sid >= nlocal) sid = nseam;
            else if (sid < p.ntx * bh) { const int tc = sid / bh; sid = tc * p.L + p.ty0 * TH + (sid - tc * bh); }
            else sid = nE + p.ty0 * p.L + (sid - p.ntx * bh);
        }
        seam_ends(p, edgeA, edgeB, sid, nE, nseam, ra[k], rb[k]);
    }
#pragma unroll
    for (int k = 0; k < SEAM_PER_THREAD; ++k) {
        todo[k] = seam_todo(ra[k], rb[k]);
        pa[k] = pb[k] = 0;
        if (todo[k]) { pa[k] = __ldcg(prov + ra[k]); pb[k] = __ldcg(prov + rb[k]); }
    }
#pragma unroll
    for (int k = 0; k < SEAM_PER_THREAD; ++k)
        if (todo[k]) gunite(prov, ra[k], rb[k], pa[k], pb[k]);
}

// ------------------------------------------------------------------------------------------------ k_final
enum { MODE_SW = 0, MODE_WOLFF = 1, MODE_LABEL = 2, MODE_FEW = 3 };

// ---- few-cluster step (S:8f row 1; reading 21): "full SW decomposition, select points, flip the distinct
// clusters these points belong to", each with probability p_flip.  k_few_seeds (one CTA, after k_seam) resolves the seed sites
// i_k = (PHILOX(seed; k, t, WSEED)[0] N) >> 32 to the roots of their global trees and enters them into a small open-addressing
// table in the workspace (-1 = empty; at least twice as many slots as seeds); k_final<MODE_FEW> looks every strip-local root's
// global root up in it and, for a selected one, draws PHILOX(seed; r, t, FLIP)[1] < T_flip.
__device__ __forceinline__ uint32_t few_slot(int root, int mask) { return ((uint32_t)root * 0x9E3779B1u >> 7) & (uint32_t)mask; }

__global__ void __launch_bounds__(256)
k_few_seeds(const Params p, const int* labels, int* __restrict__ table, int n_seeds)
{
    const int L = p.L;
    for (int i = threadIdx.x; i <= p.few_mask; i += blockDim.x) table[i] = -1;
    __syncthreads();
    for (int k = threadIdx.x; k < n_seeds; k += blockDim.x) {
        uint32_t w0, w1, w2, w3;
        philox4x32_10(p, (uint32_t)k, p.t_lo, p.t_hi, DOM_WSEED, w0, w1, w2, w3);
        const int i0 = (int)__umulhi(w0, (uint32_t)p.N);
        const int iy = i0 / L, ix = i0 - iy * L;
        const int b0 = (iy / TH * TH) * L + (ix / TW * TW);
        const int r = gfind(labels, strip_root(labels, L, i0, b0));
        uint32_t slot = few_slot(r, p.few_mask);
        while (true) {                                   // the table is never full: slots >= 2 n_seeds
            const int old = atomicCAS(&table[slot], -1, r);
            if (old == -1 || old == r) break;
            slot = (slot + 1) & (uint32_t)p.few_mask;
        }
    }
}

// is `root` a selected root, and does its draw flip it?  (The Philox call runs for selected roots only: few.)
__device__ __forceinline__ uint32_t few_flips(const Params& p, const int* __restrict__ table, int root)
{
    uint32_t slot = few_slot(root, p.few_mask);
    while (true) {
        const int e = __ldg(table + slot);
        if (e == root) break;
        if (e == -1) return 0u;
        slot = (slot + 1) & (uint32_t)p.few_mask;
    }
    uint32_t w0, w1, w2, w3;
    philox4x32_10(p, (uint32_t)root, p.t_lo, p.t_hi, DOM_FLIP, w0, w1, w2, w3);
    return w1 < p.T_flip ? 1u : 0u;
}

__device__ __forceinline__ uint32_t flip_state(const Params& p, int root)
{
    uint32_t w0, w1, w2, w3;
    philox4x32_10(p, (uint32_t)root, p.t_lo, p.t_hi, DOM_FLIP, w0, w1, w2, w3);
    return __umulhi(w0, (uint32_t)p.q);                  // uniform state in [0,q)  (S:8c.6)
}

// Shared memory of k_final: the strip's entries (node entries are rewritten in place with the FINAL value of their
// cluster: the canonical label and, in MODE_SW, the cluster's new state above bit Params::sbit -- a value >= 0) and, per
// warp, the list of the strip-local roots among the warp's own rows.
struct FinalSmem {
    int      S[TW * TH];
    uint16_t list[TW * TH];
    int      r0;
    int      ncl;                                        // global roots counted by this CTA
    int      nflip;                                      // sites flipped by this CTA (MODE_WOLFF)
};

__device__ __forceinline__ int lds_s32(uint32_t saddr)
{
    int v;
    asm volatile("ld.shared.s32 %0, [%1];" : "=r"(v) : "r"(saddr));
    return v;
}

// One CTA per strip: canonical labels (root of every site) + the new spins.
//   MODE_SW    : s_i = state drawn for the root (assign, P:55 step 3)
//   MODE_WOLFF : s_i = -s_i iff root(i) == root(seed site i0); adds |C| to *wolff_size
//   MODE_LABEL : labels only
//   MODE_FEW   : s_i = -s_i iff root(i) is a selected root whose draw is < T_flip (few-cluster step; the table of selected
//                roots comes in through the `draws` argument); adds the number of flipped sites to *wolff_size
// (1) every warp copies its rows of entries to shared memory and lists the strip-local roots among them; (2) it resolves
// each of them to the root of its global tree (a chase over entries >= 0 of other strips, which concurrently running CTAs
// may already have overwritten with final labels -- those are roots of the same tree, so the chase still ends at the
// right root) and draws one Philox state; the entry becomes the final value.  Up to here a warp touches its own rows
// only: no block barrier.  (3) every hooked node (each thread looks after its own sites) follows its references to the
// first entry >= 0 -- the strip-local root or a hooked node that is final already, both carry the final value of the
// cluster -- and takes that value.  (4) every other site is one hop from a node.
// GENR > 0: also fill the draw cache (scan_kernel.cuh) with the bond draws of step t+1 for the first GENR rows of every
// group of 4 rows of this strip: pure integer work that needs no memory, issued while the strip's entries are on their way
// from HBM.  FULL: no ragged strips (L is a multiple of TW and TH).  Q2: Ising storage (+1 / -1) of the new spins.
//
// Flags of a thread's 16 sites (4 rows x 4 columns), one bit per site in a 32-bit word: the site of row r, column j sits
// at bit 8 j + 7 - 2 r (the top bytes of a row's 4 entries, masked and shifted right by 2 r).
__device__ __forceinline__ int fin_flag_site(int b)      // bit index -> r * TW + j
{
    return (((7 - (b & 7)) >> 1) << TW_LOG) + (b >> 3);
}

#ifndef SWB_FIN_LDMODE
#define SWB_FIN_LDMODE 0
#endif
#if SWB_FIN_LDMODE == 0
#define FIN_LD(p) (*(p))
#elif SWB_FIN_LDMODE == 1
#define FIN_LD(p) __ldcg(p)
#else
#define FIN_LD(p) __ldcs(p)
#endif
// BAND: the handle works on a row band (band_kernels.cuh): the strip row is blockIdx.y + ty0.  A template parameter, because
// even this one addition in the whole-lattice kernels is measurable (k_final 0.5657 -> 0.5708 ms, k_scan 0.8637 -> 0.8656).
template <int MODE, int GENR, bool FULL, bool Q2, bool BAND = false>
__global__ void __launch_bounds__(FIN_THREADS, FIN_MIN_CTAS)
k_final(const Params p, int* labels, uint32_t* __restrict__ spins_w, Acc* __restrict__ acc,
        unsigned long long* __restrict__ wolff_size, uint32_t* __restrict__ draws)
{
    __shared__ __align__(16) FinalSmem sm;
    constexpr int R = TH / FIN_WARPS;
    static_assert(R == 4, "flag words and draw words hold the 4 rows of a warp");
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int L = p.L;
    const int x0 = blockIdx.x * TW, y0 = (blockIdx.y + (BAND ? p.ty0 : 0)) * TH;
    const int x = x0 + 4 * lane;
    const int ly0 = warp * R;
    const int base = y0 * L + x0;
    const bool colv = FULL || 4 * lane < min(TW, L - x0);
    const int nrow = FULL ? R : (colv ? max(0, min(R, L - (y0 + ly0))) : 0);   // my valid rows
    volatile int* S = sm.S;
    int* const lrow0 = labels + (size_t)(y0 + ly0) * L + x;
#if SWB_PDL
    cudaGridDependencySynchronize();
#endif
    const int l00 = ly0 * TW + 4 * lane;                 // strip-local index of my first site

    if (threadIdx.x == 0) { sm.ncl = 0; sm.nflip = 0; }
    if (MODE == MODE_WOLFF) {
        if (threadIdx.x == 0) {
            uint32_t w0, w1, w2, w3;
            philox4x32_10(p, 0u, p.t_lo, p.t_hi, DOM_WSEED, w0, w1, w2, w3);
            const int i0 = (int)__umulhi(w0, (uint32_t)p.N);
            const int iy = i0 / L, ix = i0 - iy * L;
            const int b0 = (iy / TH * TH) * L + (ix / TW * TW);
            sm.r0 = gfind(labels, strip_root(labels, L, i0, b0));
        }
    }

    // (1) my warp's rows -> shared memory; its roots -> its part of sm.list
    uint32_t hookw;                                      // flags of my hooked nodes
    uint16_t* const mylist = sm.list + warp * (R * TW);
    int nmine;                                           // roots in my warp's rows
    {
        int4 vv[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            vv[r] = make_int4(REF, REF, REF, REF);       // a site beyond a ragged edge: neither root nor hooked node
            if (FULL || r < nrow) vv[r] = FIN_LD(reinterpret_cast<const int4*>(lrow0 + (size_t)r * L));
        }
        if (GENR > 0) {
            uint32_t word = 0;
            const uint32_t c0 = (uint32_t)((y0 + ly0) * L + x) >> 1;
#pragma unroll
            for (int r = 0; r < GENR; ++r)
                if (FULL || r < nrow) word |= draw_byte(p, c0 + (uint32_t)r * ((uint32_t)L >> 1), p.u_lo, p.u_hi) << (8 * r);
            draws[draw_word_index(p, blockIdx.x, blockIdx.y + (BAND ? p.ty0 : 0), warp, lane)] = word;   // (ty = the lattice's strip row, as k_scan reads it)
        }
        uint32_t fl = 0;                                 // REF and HOOK bits of the 16 entries
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int4 v = vv[r];
            *reinterpret_cast<int4*>(&sm.S[l00 + r * TW]) = v;
            const uint32_t t = __byte_perm(__byte_perm(v.x, v.y, 0x0073), __byte_perm(v.z, v.w, 0x0073), 0x5410);
            fl |= (t & 0xC0C0C0C0u) >> (2 * r);
        }
        uint32_t rootw = ~fl & 0xAAAAAAAAu;              // REF clear
        hookw = fl & (fl << 1) & 0xAAAAAAAAu;            // REF and HOOK set
        const int cnt = __popc(rootw);
        int incl = cnt;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(FULLM, incl, o);
            if (lane >= o) incl += t;
        }
        nmine = __shfl_sync(FULLM, incl, 31);
        uint16_t* out = mylist + (incl - cnt);
        const uint32_t tag = (uint32_t)lane << 5;
        while (rootw) {                                  // entry: flag bit index | lane << 5
            const int b = 31 - __clz(rootw);
            rootw ^= 1u << b;
            *out++ = (uint16_t)(tag | (uint32_t)b);
        }
    }
    __syncwarp();
    // (2) one global resolve + one Philox draw per strip-local root, balanced over the warp.  The chase over seam-hooked
    // entries diverges (its length differs from lane to lane); the warp reconverges BEFORE the Philox draw, which would
    // otherwise be replayed once per chain length.
    int nroots = 0;
    for (int k = lane; k < nmine; k += 32) {
        const int code = mylist[k];
        const int l = ly0 * TW + fin_flag_site(code & 31) + 4 * (code >> 5);
        int v = sm.S[l];
        const int g = base + (l >> TW_LOG) * L + (l & (TW - 1));
        if (v != g) v = gfind_cached(labels, v);         // hooked by k_seam: find the root of the global tree
        __syncwarp(__activemask());
        nroots += (v == g);
        // final label and, above bit p.sbit, the new state of the cluster (labels are < 2^sbit)
        if (MODE == MODE_FEW) sm.S[l] = (int)((uint32_t)v | (few_flips(p, reinterpret_cast<const int*>(draws), v) << p.sbit));
        else sm.S[l] = MODE == MODE_SW ? (int)((uint32_t)v | (flip_state(p, v) << p.sbit)) : v;
    }
    nroots = __reduce_add_sync(FULLM, nroots);
    __syncthreads();
    if (lane == 0 && nroots) atomicAdd(&sm.ncl, nroots);
    // (3) my hooked nodes
    while (hookw) {
        const int b = 31 - __clz(hookw);
        hookw ^= 1u << b;
        const int l = l00 + fin_flag_site(b);
        int e = S[l];
        do { e = S[e & LMASK]; } while (e < 0);
        S[l] = e;
    }
    __syncthreads();

    // (4) every site
    const int r0 = MODE == MODE_WOLFF ? sm.r0 : -1;
    const int lmask = (1 << p.sbit) - 1;
    uint32_t sbase = (uint32_t)__cvta_generic_to_shared(sm.S);
    asm volatile("mov.u32 %0, %0;" : "+r"(sbase));       // keep it in a register (ptxas would recompute it at every use)
    const uint32_t sshift = (uint32_t)p.sbit - 24u, smask = 0x01010101u * ((1u << (31 - p.sbit)) - 1u);
    int nflip = 0;
    uint32_t* const srow0 = spins_w + (((size_t)(y0 + ly0) * L + x) >> 2);
#pragma unroll
    for (int r = 0; r < R; ++r) {
        if (FULL || r < nrow) {
            const int4 v = *reinterpret_cast<const int4*>(&sm.S[l00 + r * TW]);
            int ww[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
            for (int j = 0; j < 4; ++j)                  // not a node: one hop to its node, which is final
                if (ww[j] < 0) ww[j] = lds_s32(sbase + (((uint32_t)ww[j] << 2) & (uint32_t)(LMASK << 2)));
            int* const lrow = lrow0 + (size_t)r * L;
            uint32_t* const srow = srow0 + (size_t)r * (L >> 2);
            if (MODE == MODE_SW) {
                // the 4 top bytes hold the states above bit sbit - 24
                const uint32_t t = __byte_perm(__byte_perm(ww[0], ww[1], 0x0073), __byte_perm(ww[2], ww[3], 0x0073), 0x5410);
                uint32_t word = (t >> sshift) & smask;
                if (Q2) word = 0x01010101u | (word * 0xFEu);   // k=0 -> +1 (0x01), k=1 -> -1 (0xFF)
                *srow = word;
                *reinterpret_cast<int4*>(lrow) = make_int4(ww[0] & lmask, ww[1] & lmask, ww[2] & lmask, ww[3] & lmask);
            } else if (MODE == MODE_FEW) {
                // the 4 top bytes hold the flip bits above bit sbit - 24: bytes 0 / 1 -> negate the spins of the 1-bytes
                const uint32_t t = __byte_perm(__byte_perm(ww[0], ww[1], 0x0073), __byte_perm(ww[2], ww[3], 0x0073), 0x5410);
                const uint32_t word = (t >> sshift) & smask & 0x01010101u;
                if (word) {
                    const uint32_t m = word * 0xFFu, old = *srow;
                    *srow = __vneg4(old & m) | (old & ~m);
                    nflip += __popc(word);
                }
                *reinterpret_cast<int4*>(lrow) = make_int4(ww[0] & lmask, ww[1] & lmask, ww[2] & lmask, ww[3] & lmask);
            } else {
                *reinterpret_cast<int4*>(lrow) = make_int4(ww[0], ww[1], ww[2], ww[3]);
            }
            if (MODE == MODE_WOLFF) {
                const uint32_t m = (ww[0] == r0 ? 0xFFu : 0u) | (ww[1] == r0 ? 0xFF00u : 0u) |
                                   (ww[2] == r0 ? 0xFF0000u : 0u) | (ww[3] == r0 ? 0xFF000000u : 0u);   // bytes to negate
                if (m) {
                    const uint32_t old = *srow;
                    *srow = __vneg4(old & m) | (old & ~m);
                    nflip += __popc(m) >> 3;
                }
            }
        }
    }
    // one 64-bit atomic per CTA, spread over ACC_PARTS addresses in different 128-byte lines: tens of thousands of atomics
    // on ONE address serialise in a single L2 slice and stall the whole kernel (measured: 0.71 -> 0.50 ms at beta = 0.5)
    if (threadIdx.x == 0 && sm.ncl)
        atomicAdd(&acc->part[(blockIdx.x + 5 * blockIdx.y) & (ACC_PARTS - 1)].n_clusters, (unsigned long long)sm.ncl);
    if (MODE == MODE_WOLFF || MODE == MODE_FEW) {
        nflip = __reduce_add_sync(FULLM, nflip);
        if (lane == 0 && nflip) atomicAdd(&sm.nflip, nflip);
        __syncthreads();
        if (threadIdx.x == 0 && sm.nflip) atomicAdd(wolff_size, (unsigned long long)sm.nflip);
    }
}

}  // namespace swb
