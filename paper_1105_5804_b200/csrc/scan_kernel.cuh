// scan_kernel.cuh -- k_scan: bond activation (P:53 step 1, Eq. 7) fused with strip-local labelling.
// Included by label_kernels.cuh (uses its forest helpers nm_find / nm_root4 and the `prov` encoding).
//
// One warp per TW x TH strip, lane -> 4 consecutive columns, rows in sequence.  A "node" is a site that names a run: the
// first site of a part of a horizontal run (the part inside one lane, or inside two neighbouring lanes) that has no active
// north bond from the row above.  Every other site adopts the name carried by the leftmost contact of its part with the row
// above, so every name is a node.  Wherever two names meet that are not known to be equal -- a contact whose carried name
// differs from the adopted one, or a run that continues from the left lane into a fully bonded lane -- a flag bit is set;
// the flagged site positions are collected every 8 rows and their names united, 32 pairs at a time (all lanes busy), in
// the strip's forest.  Names never depend on the forest, so the row loop has no divergent part.
//
// The kernel is bound by the integer ALU pipe (LOP3, PRMT, ISETP, SEL, SHF: one warp instruction per 2 clocks per
// sub-partition; measured, profiles/r02_README.md), so the row loop is written to keep work OFF that pipe:
//   - names are strip-local site indices (< TW*TH = 4096) kept as 16-bit halves, two per register (P01/P23 = names
//     carried by the 4 sites of the previous row, l01/l23 = names of this row); which name a site takes inside its lane is
//     a function of 8 bits -- the lane's 4 east bonds and the 4 north bonds from the row above -- so it comes from a
//     256-entry table of byte-permutation selectors: 4 PRMT name the 4 sites;
//   - a run that crosses into the next lane is resolved between the two neighbours only: two shuffles carry the suffix name
//     of the left lane and the prefix name of the right lane plus flag bits; masks from the same table entry decide with one
//     LOP3 each whether the lane's prefix / suffix part takes the neighbour's name (predicated PRMTs, selectors from a second
//     small table).  No ballots, no bit scans.  A fully bonded lane keeps its own name and flags the link instead;
//   - "is this half-word non-zero" for the 4 mismatch tests is an add that carries out of the 12-bit name, on the
//     multiply-add pipe; the 4 carries are gathered with a multiply-high; flag words are accumulated with multiply-adds.
#pragma once
#include "common.cuh"

namespace swb {

static_assert(TW * TH <= 4096, "names are 12-bit strip-local site indices");

// ---------------------------------------------------------------------------------------------------- host/device helpers
// PRMT reads the 4 selector nibbles of s[15:0] only (every nibble here is < 8: plain byte select); the upper half of a
// selector word is free for other table data.  The host versions serve tests/host/scan_row_check.cu.
#define SWB_HD __host__ __device__ __forceinline__
SWB_HD uint32_t prmt(uint32_t a, uint32_t b, uint32_t s)
{
#ifdef __CUDA_ARCH__
    uint32_t d;
    asm("prmt.b32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(s));
    return d;
#else
    const uint64_t ab = ((uint64_t)b << 32) | a;
    uint32_t d = 0;
    for (int i = 0; i < 4; ++i) d |= (uint32_t)((ab >> (8 * ((s >> (4 * i)) & 7))) & 0xFF) << (8 * i);
    return d;
#endif
}
SWB_HD uint32_t mulhi_u32(uint32_t a, uint32_t b)
{
#ifdef __CUDA_ARCH__
    return __umulhi(a, b);
#else
    return (uint32_t)(((uint64_t)a * b) >> 32);
#endif
}

// ---------------------------------------------------------------------------------------------------- tables
// A half h in [0,4) of a register pair (a, b) seen by PRMT: 0 = a.lo, 1 = a.hi, 2 = b.lo, 3 = b.hi.
constexpr uint32_t lut_half(int h) { return (uint32_t)(((2 * h + 1) << 4) | (2 * h)); }
constexpr uint32_t lut_sel(int hlo, int hhi) { return lut_half(hlo) | (lut_half(hhi) << 8); }

// Flag bits in the upper halves of the table words (the lower halves are PRMT selectors)
constexpr uint32_t F_LK = 1u << 16;      // a[0]: my east bond into the next lane is active (sent to the right neighbour)
constexpr uint32_t F_LC = 1u << 17;      // a[0]: ... and my suffix part has a contact
constexpr uint32_t F_CP = 1u << 20;      // a[1]: my prefix part has a contact (sent to the left neighbour)
                                         // a[1] bits 16,17: link-flag masks against the left neighbour's F_LK, F_LC
                                         // a[2] bits 16,17: prefix-substitution masks against F_LK, F_LC; bit 20: suffix-
                                         //                  substitution mask against the right neighbour's F_CP
                                         // a[3] bits 16..19: north contacts of sites 0..3

struct ScanLut {
    uint32_t a[256][4];    // index: bit 2j = E_j (east bond site j -> j+1, E_3 into the next lane), bit 2j+1 = north bond from
                           // the previous row into site j: (bond byte of this row & 0x55) | (bond byte of the previous & 0xAA)
    uint32_t b[22][4];     // index: bond byte & 0x15 (E_0, E_1, E_2): which sites belong to the prefix / suffix part
};

constexpr ScanLut make_scan_lut()
{
    ScanLut t{};
    for (int i = 0; i < 256; ++i) {
        const bool E0 = i & 1, E1 = i & 4, E2 = i & 16, E3 = i & 64;
        const int np = ((i >> 1) & 1) | (((i >> 3) & 1) << 1) | (((i >> 5) & 1) << 2) | (((i >> 7) & 1) << 3);
        int s[4] = {0, 0, 0, 0};                         // first site of each site's part (run inside the lane)
        s[1] = E0 ? 0 : 1;
        s[2] = E1 ? s[1] : 2;
        s[3] = E2 ? s[2] : 3;
        int lc[4] = {-1, -1, -1, -1};                    // leftmost contact of the part, -1: none
        for (int j = 0; j < 4; ++j)
            for (int k = 3; k >= 0; --k)
                if (s[k] == s[j] && ((np >> k) & 1)) lc[j] = k;
        // X = prmt(P01, P23, selX): the contact names that sites 0 and 1 may take
        const uint32_t selX = lut_sel(lc[0] < 0 ? 0 : lc[0], lc[1] < 0 ? 0 : lc[1]);
        // l01 = prmt(X, NEW01, selL01): contact name, else a new node named by the part's first site
        const uint32_t selL01 = lut_sel(lc[0] < 0 ? 2 : 0, lc[1] < 0 ? 2 + s[1] : 1);
        // W = prmt(P23, NEW23, selW): names of sites 2 / 3 if they start a part (s == own index)
        const int wlo = s[2] != 2 ? 0 : (lc[2] < 0 ? 2 : lc[2] - 2);
        const int whi = (np & 8) ? 1 : 3;
        const uint32_t selW = lut_sel(wlo, whi);
        // l23 = prmt(W, l01, selL23): a site whose part starts at 0 or 1 takes l1
        const uint32_t selL23 = lut_sel(s[2] == 2 ? 0 : 3, s[3] == 3 ? 1 : (s[3] == 2 ? 0 : 3));
        const bool full = E0 && E1 && E2, cp = lc[0] >= 0, cs = lc[3] >= 0;
        t.a[i][0] = selX | (E3 ? F_LK : 0u) | (E3 && cs ? F_LC : 0u);
        // link flag (fully bonded lanes only): the run continues from the left lane and this lane keeps its own name --
        // unless the left part has no contact and this lane has one (then the left part takes this lane's name)
        t.a[i][1] = selL01 | (cp ? F_CP : 0u) | (full && !cp ? F_LK : 0u) | (full ? F_LC : 0u);
        // the prefix part takes the left suffix name if the link is active and (the left part has a contact or mine has
        // none); the suffix part takes the right prefix name if my link is active, mine has no contact and the right has one
        t.a[i][2] = selW | (!full && !cp ? F_LK : 0u) | (!full ? F_LC : 0u) | (E3 && !cs ? F_CP : 0u);
        t.a[i][3] = selL23 | ((uint32_t)np << 16);
    }
    for (int i = 0; i < 22; ++i) {
        const bool E0 = i & 1, E1 = i & 4, E2 = i & 16;
        int s[4] = {0, 0, 0, 0};
        s[1] = E0 ? 0 : 1;
        s[2] = E1 ? s[1] : 2;
        s[3] = E2 ? s[2] : 3;
        // l' = prmt(l, nb, sel): own halves 0, 1; the neighbour's name is the low half of nb = half 2
        t.b[i][0] = lut_sel(2, s[1] == 0 ? 2 : 1);                              // prefix part, sites 0 1
        t.b[i][1] = lut_sel(s[2] == 0 ? 2 : 0, s[3] == 0 ? 2 : 1);              // prefix part, sites 2 3
        t.b[i][2] = lut_sel(s[0] == s[3] ? 2 : 0, s[1] == s[3] ? 2 : 1);        // suffix part, sites 0 1
        t.b[i][3] = lut_sel(s[2] == s[3] ? 2 : 0, 2);                           // suffix part, sites 2 3
    }
    return t;
}

// ---------------------------------------------------------------------------------------------------- one row of one lane
// Part 1: names from the lane's own bonds and contacts, and the two messages to the neighbouring lanes:
//   to the right: suffix name | F_LK, F_LC      to the left: prefix name | F_CP
SWB_HD void row_local(const uint32_t A[4], uint32_t P01, uint32_t P23, uint32_t NEW01, uint32_t NEW23,
                      uint32_t& l01, uint32_t& l23, uint32_t& to_right, uint32_t& to_left)
{
    const uint32_t X = prmt(P01, P23, A[0]);
    l01 = prmt(X, NEW01, A[1]);
    const uint32_t W = prmt(P23, NEW23, A[2]);
    l23 = prmt(W, l01, A[3]);
    to_right = prmt(l23, A[0], 0x7632);                  // l3 | upper half of A[0]
    to_left = prmt(l01, A[1], 0x7610);                   // l0 | upper half of A[1]
}

// Part 2: substitute the neighbours' names where the table masks say so; returns the link flag (0 / non-zero in bits
// 16,17).  left_ok = F_LK | F_LC, or 0 for the first lane of the strip (no left neighbour).
SWB_HD uint32_t row_final(const uint32_t A[4], const uint32_t B[4], uint32_t from_left, uint32_t from_right,
                          uint32_t left_ok, uint32_t& l01, uint32_t& l23)
{
    const bool subP = (from_left & A[2] & left_ok) != 0u;
    const bool subS = (from_right & A[2] & F_CP) != 0u;
    if (subP) { l01 = prmt(l01, from_left, B[0]); l23 = prmt(l23, from_left, B[1]); }
    if (subS) { l01 = prmt(l01, from_right, B[2]); l23 = prmt(l23, from_right, B[3]); }
    return from_left & A[1] & left_ok;
}

// The 4 mismatch flags of the row in bits 16..19: site j carries a contact (north bond from the row above) whose name P_j
// differs from the name l_j it has taken.  Names are < 4096: x + 0x0FFF carries into bit 12 iff x != 0.
SWB_HD uint32_t row_mismatch(const uint32_t A[4], uint32_t P01, uint32_t P23, uint32_t l01, uint32_t l23)
{
    const uint32_t t01 = (P01 ^ l01) + 0x0FFF0FFFu;                      // bits 12, 28: sites 0, 1
    const uint32_t t23 = (P23 ^ l23) * 4u + 0x3FFC3FFCu;                 // bits 14, 30: sites 2, 3
    const uint32_t r = (t01 & 0x10001000u) | (t23 & 0x40004000u);
    // gather bits 12, 28, 14, 30 into bits 0, 1, 2, 3 of the high word: 2^20 moves 12 -> 0 and 14 -> 2, 2^5 moves 28 -> 1 and
    // 30 -> 3; the cross terms land on bits 16, 18 (shifted out below) or in the low word
    const uint32_t nib = mulhi_u32(r, (1u << 20) | (1u << 5));
    return (nib << 16) & A[3];
}

__device__ const ScanLut d_scan_lut = make_scan_lut();

// ---------------------------------------------------------------------------------------------------- device helpers
// d <- 2 d + [u >= T] for T != 0: the carry of u + (2^32 - T) shifted into d.  An add with carry-out (ALU pipe) and an
// add with carry-in (ptxas issues it as IMAD.X on the multiply-add pipe): no compare, select or shift.
__device__ __forceinline__ void shift_in_ge(uint32_t& d, uint32_t u, uint32_t negT)
{
    asm("{\n\t.reg .u32 t;\n\tadd.cc.u32 t, %1, %2;\n\taddc.u32 %0, %0, %0;\n\t}" : "+r"(d) : "r"(u), "r"(negT));
}

// a * b + c on the multiply-add pipe (the compiler would turn a multiply by a power of two into an ALU shift)
__device__ __forceinline__ uint32_t mad_lo(uint32_t a, uint32_t b, uint32_t c)
{
    uint32_t d;
    asm("mad.lo.u32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
    return d;
}
__device__ __forceinline__ uint32_t mad_hi(uint32_t a, uint32_t b, uint32_t c)
{
    uint32_t d;
    asm("mad.hi.u32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
    return d;
}

// Draw byte of the 4 sites whose first pair has Philox counter c0, at step (t_lo, t_hi): bit 2j = [east draw of site j
// >= T], bit 2j+1 = [north draw >= T] (S:8c.3: u(i,d,t) = PHILOX(seed; i>>1, t, BOND)[2(i&1)+d]).  A pure function of
// (seed, t, site, T): k_final can compute it one sweep ahead (draw cache, see k_final) and k_scan<SRC_DRAWS> only reads it.
__device__ __forceinline__ uint32_t draw_byte(const Params& p, uint32_t c0, uint32_t t_lo, uint32_t t_hi)
{
    uint32_t a0, a1, a2, a3, b0, b1, b2, b3;
    philox4x32_10(p, c0, t_lo, t_hi, DOM_BOND, a0, a1, a2, a3);
    philox4x32_10(p, c0 + 1, t_lo, t_hi, DOM_BOND, b0, b1, b2, b3);
    uint32_t d = 0;                                      // the last draw first, it ends up in bit 7
    shift_in_ge(d, b3, p.negT); shift_in_ge(d, b2, p.negT); shift_in_ge(d, b1, p.negT); shift_in_ge(d, b0, p.negT);
    shift_in_ge(d, a3, p.negT); shift_in_ge(d, a2, p.negT); shift_in_ge(d, a1, p.negT); shift_in_ge(d, a0, p.negT);
    return d;
}

// The lane's bond byte for row y: bit 2j = east bond of site j, bit 2j+1 = north bond of site j (the packed-bond
// format of include/swb200.h), for the 4 sites whose spins are w; e = spins of the east neighbours, n = of the north;
// d = their draw byte.
template <bool ISING>
__device__ __forceinline__ uint32_t bond_byte(const Params& p, uint32_t d, uint32_t w, uint32_t e, uint32_t n,
                                              uint32_t& ce, uint32_t& cn)
{
    // ce / cn: one bit per site (bit 8j+1 / 8j+2) that tells whether the east / north bond of site j is UNsatisfied (Ising)
    // or satisfied (Potts); the caller adds them up byte-wise over the rows of a strip (the fused energy count)
    uint32_t eq;                                         // bit 8j+1: s_j == s_east, bit 8j+2: s_j == s_north
    if (ISING) {                                         // bytes 0x01 / 0xFF: equal <=> bit 1 (and bit 2) of the xor is 0
        ce = (w ^ e) & 0x02020202u;
        cn = (w ^ n) & 0x04040404u;
        eq = ~(ce | cn) & 0x06060606u;
    } else {
        ce = __vcmpeq4(w, e) & 0x02020202u;
        cn = __vcmpeq4(w, n) & 0x04040404u;
        eq = ce | cn;
    }
    // gather the 4 bit pairs (8j+1, 8j+2) into bits (2j, 2j+1) of the high word; the cross terms of the product land on
    // distinct bits below 32 or above bit 7 of the high word (no carries)
    // p.dmask = 0xFF, or 0 if T = 0 (then u >= T always, but u + 2^32 never carries)
    return __umulhi(eq, 0x82082000u) & ~d & p.dmask;     // 2^31 + 2^25 + 2^19 + 2^13
}

// sum of the 4 bytes of x
__device__ __forceinline__ uint32_t byte_sum(uint32_t x)
{
    x = (x & 0x00FF00FFu) + ((x >> 8) & 0x00FF00FFu);
    return (x + (x >> 16)) & 0xFFFFu;
}

// Draw cache (workspace): one 32-bit word per lane and group of 4 rows of a strip, byte r = draw byte of row 4g + r:
// word index ((ty * ntx + tx) * (TH / 4) + g) * 32 + lane.  Written by k_final<MODE_SW> for step t+1 (its warp g owns rows
// 4g..4g+3), read by k_scan<SRC_DRAWS> of the next sweep.
__device__ __forceinline__ size_t draw_word_index(const Params& p, int tx, int ty, int g, int lane)
{
    return ((size_t)(ty * p.ntx + tx) * (TH / 4) + g) * 32 + lane;
}

// ---------------------------------------------------------------------------------------------------- unions
// Queue entries: bits 0..11 = strip-local position p of a flagged site, QEAST set: unite the names of p and of its west
// neighbour p - 1 (link flag), else of p and of the site above it, p - TW (mismatch flag).  Names are read back from the
// forest array: entry of a site = the name it took (a node) or, for a node, its parent.
constexpr uint32_t QEAST = 0x8000u;
#ifndef SWB_UNITE_V2
#define SWB_UNITE_V2 1
#endif
#ifndef SWB_DRAIN_SCAN
#define SWB_DRAIN_SCAN 1
#endif
// Queue capacity per warp: a drain appends all flagged sites of 8 rows at once when they fit (the usual case: about 100
// at beta_c), else 32 at a time.
constexpr int QCAP = SCAN_WARPS >= 8 ? 384 : 64;

// Unite one queued pair per lane, hooking the larger root under the smaller and writing every hook through to `prov`.
// 3-phase protocol, no atomics (the forest belongs to this warp): (1) all lanes find the roots of their two names, the two
// chases in lockstep, and point the two names directly at their roots (the same names keep coming back while a cluster
// grows down the strip) -- nobody hooks, so a root stays a root; (2) hook with a plain store -- lanes hooking the same
// root collide, one store wins; (3) re-read: losers retry from the new roots.
__device__ __forceinline__ void unite_batch(volatile uint16_t* nm, bool have, uint32_t code, int* prov, int base, int L)
{
    int ua = 0, ub = 0;
    if (have) {
        const int pos = (int)(code & 0x0FFFu);
        ua = nm[pos];
        ub = nm[pos - ((code & QEAST) ? 1 : TW)];
    }
    while (__any_sync(FULLM, have)) {
        if (have) {
#if SWB_UNITE_V2
            const int a0 = ua, b0 = ub;
            int pa = nm[ua], pb = nm[ub];
            ua = pa; ub = pb;                            // one unconditional hop (a root points to itself): measured -1.6 %
            pa = nm[ua]; pb = nm[ub];
            while ((pa ^ ua) | (pb ^ ub)) {
                ua = pa; ub = pb;
                pa = nm[ua]; pb = nm[ub];
            }
            if (a0 != ua) nm[a0] = (uint16_t)ua;
            if (b0 != ub) nm[b0] = (uint16_t)ub;
#else
            ua = nm_find(nm, ua);
            ub = nm_find(nm, ub);
#endif
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

// Collect the flagged sites of the lanes' flag words into the warp's queue and unite them 32 at a time.  Bit b of `flags`
// stands for the strip-local position pos0 - (b >> sh) * TW + (b & ((1 << sh) - 1)) (sh = 2: 4 mismatch flags per row, the
// newest row in bits 0..3; sh = 0: one link flag per row) | tag.  If all of them fit into the queue, a warp scan of the
// per-lane counts gives every lane its slots and it appends its own entries; else every round each lane that still has a
// flag appends one and full batches are united on the way.
__device__ __forceinline__ void drain_flags(uint32_t flags, int sh, int pos0, uint32_t tag, volatile uint16_t* q, int& qn,
                                            volatile uint16_t* nm, int* prov, int base, int L, int lane, unsigned lt)
{
    if (SWB_DRAIN_SCAN && QCAP >= 128) {                 // (a 64-entry queue never takes 8 rows at once: skip the scan)
        const int cnt = __popc(flags);
        int incl = cnt;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(FULLM, incl, o);
            if (lane >= o) incl += t;
        }
        const int total = __shfl_sync(FULLM, incl, 31);
        if (total == 0) return;
        if (total <= QCAP - qn) {
            volatile uint16_t* out = q + qn + (incl - cnt);
            while (flags) {
                const int b = 31 - __clz(flags);
                flags ^= 1u << b;
                *out++ = (uint16_t)((uint32_t)(pos0 - ((b >> sh) << TW_LOG) + (b & ((1 << sh) - 1))) | tag);
            }
            qn += total;
            __syncwarp();                                // queue entries and forest rows visible to the whole warp
            while (qn >= 32) {
                qn -= 32;
                unite_batch(nm, true, q[qn + lane], prov, base, L);
            }
            __syncwarp();                                // queue slots read before they are overwritten
            return;
        }
    }
    while (true) {
        const bool has = flags != 0u;
        const unsigned Bm = __ballot_sync(FULLM, has);
        if (Bm == 0u) break;
        if (has) {
            const int b = 31 - __clz(flags);
            flags ^= 1u << b;
            const int pos = pos0 - ((b >> sh) << TW_LOG) + (b & ((1 << sh) - 1));
            q[qn + __popc(Bm & lt)] = (uint16_t)((uint32_t)pos | tag);
        }
        qn += __popc(Bm);
        __syncwarp();
        while (qn >= 32) {
            qn -= 32;
            unite_batch(nm, true, q[qn + lane], prov, base, L);
        }
        __syncwarp();
    }
}

// ---------------------------------------------------------------------------------------------------- k_scan
#ifndef SWB_SCAN_UNROLL
#define SWB_SCAN_UNROLL 1
#endif
constexpr int SCAN_UNROLL = SWB_SCAN_UNROLL;

struct ScanSmem {
    uint16_t nm[SCAN_WARPS][TW * TH];                    // the strips' forests
    uint4    la[256];                                    // naming tables
    uint4    lb[22];
    uint16_t q[SCAN_WARPS][QCAP];                        // queues of flagged sites
    uint8_t  e3[SCAN_WARPS][TH];                         // bond byte of the strip's last lane, row by row (bit 6 leaves the strip)
#ifdef SWB_SCAN_PAD
    uint8_t  pad[SWB_SCAN_PAD];
#endif
};

// SRC_PHILOX: read spins, draw bonds (a1).  SRC_DRAWS: read spins and the draw cache k_final filled one sweep ahead (the
// same bonds, the Philox work done elsewhere).  SRC_BONDS: read packed bonds (sw_label).  Writes the provisional labels
// (`prov`, see label_kernels.cuh) and the edge arrays, and adds the number of active bonds to the sweep counters.
// FULLW: L is a multiple of TW, every strip has all 32 lanes (no ragged right edge; the predicates fold away).
enum { SRC_PHILOX = 0, SRC_BONDS = 1, SRC_DRAWS = 2 };
template <int SRC, bool ISING, bool FULLW, bool BAND = false>    // BAND: strip row = blockIdx.y + ty0 (see k_final)
#ifndef SWB_SCAN_RES_WARPS
#define SWB_SCAN_RES_WARPS 24
#endif
__global__ void __launch_bounds__(SCAN_THREADS, SWB_SCAN_RES_WARPS / SCAN_WARPS)    // 24 warps per SM (shared memory): up to 85 registers
k_scan(const Params p, const uint32_t* __restrict__ spins_w, const uint8_t* __restrict__ bonds_in,
       const uint32_t* __restrict__ draws, int* prov, int* __restrict__ edgeA, int* __restrict__ edgeB,
       Acc* __restrict__ acc)
{
    constexpr bool FROM_BONDS = SRC == SRC_BONDS;
    extern __shared__ __align__(16) unsigned char s_raw[];   // ScanSmem: 37.9 KB with SCAN_WARPS = 4; dynamic because a SCAN_WARPS = 8 build exceeds the 48 KB of a static allocation
    ScanSmem& sm = *reinterpret_cast<ScanSmem*>(s_raw);
    uint4* const s_la = sm.la;
    uint4* const s_lb = sm.lb;
    for (int i = threadIdx.x; i < 256; i += SCAN_THREADS)
        s_la[i] = make_uint4(d_scan_lut.a[i][0], d_scan_lut.a[i][1], d_scan_lut.a[i][2], d_scan_lut.a[i][3]);
    for (int i = threadIdx.x; i < 22; i += SCAN_THREADS)
        s_lb[i] = make_uint4(d_scan_lut.b[i][0], d_scan_lut.b[i][1], d_scan_lut.b[i][2], d_scan_lut.b[i][3]);
    __syncthreads();                                     // the only block-wide barrier
#if SWB_PDL == 2
    cudaGridDependencySynchronize();                     // (the tables do not depend on the preceding kernels)
#endif

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int tx = blockIdx.x * SCAN_WARPS + warp, ty = blockIdx.y + (BAND ? p.ty0 : 0);
    if (tx >= p.ntx) return;
    uint16_t* nm = sm.nm[warp];
    volatile uint16_t* vnm = nm;
    volatile uint16_t* q = sm.q[warp];
    uint8_t* const s_e3 = sm.e3[warp];
    const int L = p.L, Lw = L >> 2;
    const int x0 = tx * TW, y0 = ty * TH;
    const int tw_eff = FULLW ? TW : min(TW, L - x0), th_eff = min(TH, L - y0);
    const int x = x0 + 4 * lane;
    const bool colv = FULLW || 4 * lane < tw_eff;
    const int last_lane = (tw_eff >> 2) - 1;             // lane that owns the strip's last column
    const bool is_last = lane == last_lane;
    const int base = y0 * L + x0;
    const int xw = x >> 2;
    const int xew = ((x + 4 == L) ? 0 : x + 4) >> 2;     // east halo word of the last lane (periodic)
    const unsigned lt = lanemask_lt();
    // the east bond that leaves the strip is dropped from the lane's bond byte; lanes beyond a ragged edge have no bonds
    const uint32_t gmask = !colv ? 0u : is_last ? 0xBFu : 0xFFu;
    const uint32_t left_ok = lane ? (F_LK | F_LC) : 0u;  // the first lane has no left neighbour

    // spin words of rows y, y+1, y+2 (w*) and the east halo words of the last lane (h*); row index L wraps to 0
    uint32_t w0 = 0, w1 = 0, w2 = 0, h0 = 0, h1 = 0, h2 = 0;
    const int yend = y0 + th_eff;                        // north neighbour row of the strip's last row
    const int row_halo = (yend == L ? 0 : yend) * Lw;    // its word offset
    const int xws = colv ? xw : (x0 >> 2);               // lanes beyond a ragged edge read a valid word (their bonds are masked)
    if (!FROM_BONDS) {
        w0 = spins_w[(size_t)y0 * Lw + xws];
        if (is_last) h0 = spins_w[(size_t)y0 * Lw + xew];
        const int r1 = th_eff > 1 ? (y0 + 1) * Lw : row_halo;
        w1 = spins_w[r1 + xws];
        if (is_last) h1 = spins_w[r1 + xew];
        if (th_eff > 1) {
            const int r2 = th_eff > 2 ? (y0 + 2) * Lw : row_halo;
            w2 = spins_w[r2 + xws];
            if (is_last) h2 = spins_w[r2 + xew];
        }
    }

    uint32_t P01 = 0, P23 = 0;                           // names carried by the previous row's sites
    uint32_t Gn = 0;                                     // north bonds of the previous row (bits 1,3,5,7 of its bond byte)
    uint32_t NEW01 = (uint32_t)(4 * lane) * 0x00010001u + 0x00010000u;      // own names of sites 0,1 / 2,3 of this row
    uint32_t NEW23 = NEW01 + 0x00020002u;
    uint32_t nact = 0;
    uint32_t acc_e = 0, acc_n = 0, acc_m = 0;            // byte-wise sums for the fused energy / magnetisation count
    int qn = 0;                                          // queued entries (warp-uniform)
    uint32_t fl = 0;                                     // mismatch flags, 4 per row, the newest row in bits 0..3
    uint32_t fe = 0;                                     // link flags, 1 per row, the newest row in bit 0

    // running per-row quantities: Philox counter of the lane's first pair, global index of the lane's first site, pointer
    // to the lane's spin word of the row to prefetch (ly + 3)
    uint32_t c0 = (uint32_t)(y0 * L + x) >> 1;
    int gi = y0 * L + x;
    const uint32_t* pw = spins_w + (size_t)(y0 + 3) * Lw + xws;   // the lane's word of the row to prefetch; halo: + dxe
    const uint32_t* const pw_halo = spins_w + row_halo + xws;
    const int dxe = xew - xws;
    uint32_t dw = 0;                                     // draw bytes of the rows 4g..4g+3 (SRC_DRAWS)
    const uint32_t* pdw = draws + (SRC == SRC_DRAWS ? draw_word_index(p, tx, ty, 0, lane) : 0);
    uint32_t G = 0;                                      // the lane's bond byte of the current row

    // (Computing the bond byte, or only its Philox draws, one row ahead of the naming chain -- software pipelining inside
    // the warp -- was measured slower: 0.88 -> 0.91 / 1.01 ms; the other warps of the sub-partition hide that latency.)
#pragma unroll SCAN_UNROLL
    for (int ly = 0; ly < th_eff; ++ly) {
        if (!FROM_BONDS) {
            uint32_t d;
            if (SRC == SRC_DRAWS && (ly & 3) == 0) { dw = *pdw; pdw += 32; }
            if (SRC == SRC_DRAWS && (ly & 3) < GEN_ROWS) d = __byte_perm(dw, 0u, 0x4440u | (uint32_t)(ly & 3));
            else d = draw_byte(p, c0, p.t_lo, p.t_hi);
            uint32_t w3 = 0, h3 = 0;                     // prefetch row y+3 (the last one is the north halo row)
            if (ly + 3 <= th_eff) {
                const uint32_t* const q3 = ly + 3 < th_eff ? pw : pw_halo;
                w3 = *q3;
                if (is_last) h3 = q3[dxe];
            }
            pw += Lw;
            uint32_t wnext = __shfl_down_sync(FULLM, w0, 1);
            if (is_last) wnext = h0;
            const uint32_t east = __funnelshift_r(w0, wnext, 8);
            uint32_t ce, cn;
            G = bond_byte<ISING>(p, d, w0, east, w1, ce, cn);
            // energy and magnetisation of the configuration this sweep starts from, for free (Eq. 1; BJ north_star (5)):
            // the (un)satisfied-bond bits are here already; they are added up byte-wise (2 / 4 per bond, at most TH = 32 rows:
            // no byte overflows) with adds on the multiply-add pipe and evaluated once per strip
            acc_e = mad_lo(ce, 1u, acc_e);
            acc_n = mad_lo(cn, 1u, acc_n);
            if (ISING) acc_m = mad_lo(w0 & 0x02020202u, 1u, acc_m);       // a byte 0xFF (spin -1) adds 2
            c0 += (uint32_t)L >> 1;
            w0 = w1; w1 = w2; w2 = w3; h0 = h1; h1 = h2; h2 = h3;
        } else {
            G = colv ? bonds_in[(size_t)gi >> 2] : 0u;
        }
        // the bond that leaves the strip to the east is remembered for the edge arrays and dropped here
        if (is_last) s_e3[ly] = (uint8_t)G;
        G &= gmask;
        nact += __popc(G);

        // ---- names of this row's sites ----------------------------------------------------------------------
        const uint4 A4 = s_la[(G & 0x55u) | Gn];
        const uint4 B4 = s_lb[G & 0x15u];
        const uint32_t A[4] = {A4.x, A4.y, A4.z, A4.w}, B[4] = {B4.x, B4.y, B4.z, B4.w};
        uint32_t l01, l23, to_right, to_left;
        row_local(A, P01, P23, NEW01, NEW23, l01, l23, to_right, to_left);
        const uint32_t from_left = __shfl_up_sync(FULLM, to_right, 1);
        const uint32_t from_right = __shfl_down_sync(FULLM, to_left, 1);
        const uint32_t link = row_final(A, B, from_left, from_right, left_ok, l01, l23);
        // link flag -> fe = 2 fe + [link != 0]: (link + 0x30000) >> 18 on the multiply-add pipe
        fe = mad_hi(link + 0x00030000u, 1u << 14, fe + fe);
        // mismatch flags -> fl = 16 fl + flags
        fl = mad_hi(row_mismatch(A, P01, P23, l01, l23), 1u << 16, mad_lo(fl, 16u, 0u));

        // the row's entries in the forest (a new node's name is its own index, i.e. it starts as a root) and in `prov`
        *reinterpret_cast<uint2*>(nm + ly * TW + 4 * lane) = make_uint2(l01, l23);
        if (colv) {
            const uint32_t z01 = l01 ^ NEW01, z23 = l23 ^ NEW23;
            int4 g;
            g.x = (z01 & 0xFFFFu) ? (int)prmt(l01, 0x80000000u, 0x7610) : gi;
            g.y = (z01 >> 16) ? (int)prmt(l01, 0x80000000u, 0x7632) : gi + 1;
            g.z = (z23 & 0xFFFFu) ? (int)prmt(l23, 0x80000000u, 0x7610) : gi + 2;
            g.w = (z23 >> 16) ? (int)prmt(l23, 0x80000000u, 0x7632) : gi + 3;
            *reinterpret_cast<int4*>(prov + (size_t)gi) = g;
        }

        if ((ly & 7) == 7) {                             // unite the names of the flagged sites of the last 8 rows
            __syncwarp();
            drain_flags(fl, 2, ly * TW + 4 * lane, 0u, q, qn, vnm, prov, base, L, lane, lt);
            fl = 0;
        }

        P01 = l01; P23 = l23;
        Gn = G & 0xAAu;
        NEW01 += (uint32_t)TW * 0x00010001u;
        NEW23 += (uint32_t)TW * 0x00010001u;
        gi += L;
    }

    __syncwarp();
    drain_flags(fl, 2, (th_eff - 1) * TW + 4 * lane, 0u, q, qn, vnm, prov, base, L, lane, lt);    // rows since the last drain
    drain_flags(fe, 0, (th_eff - 1) * TW + 4 * lane, QEAST, q, qn, vnm, prov, base, L, lane, lt);  // link flags of all rows
    __syncwarp();
    if (qn > 0) {
        const bool have = lane < qn;
        unite_batch(vnm, have, have ? q[lane] : 0u, prov, base, L);
    }
    __syncwarp();

    // ---- edge arrays: strip-local roots of the sites on the four edges ----------------------------------------------
    {
        const int nE = p.ntx * L;
        const uint32_t northm = G;                       // bond byte of the last row: its north bonds leave the strip
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
            n.x = (northm & 0x02u) ? strip_gidx(base, L, n0) : -1;
            n.y = (northm & 0x08u) ? strip_gidx(base, L, n1) : -1;
            n.z = (northm & 0x20u) ? strip_gidx(base, L, n2) : -1;
            n.w = (northm & 0x80u) ? strip_gidx(base, L, n3) : -1;
            *reinterpret_cast<int4*>(edgeB + (size_t)nE + (size_t)ty * L + x) = s;
            *reinterpret_cast<int4*>(edgeA + (size_t)nE + (size_t)ty * L + x) = n;
        }
        // first column -> rootW, last column -> rootE: lane i takes row i
        uint32_t e3 = 0;
        if (lane < th_eff) {
            e3 = s_e3[lane] & 0x40u;
            int w = lane * TW, e = lane * TW + tw_eff - 1, w2 = w, e2 = e;
            nm_root4(vnm, w, e, w2, e2);
            edgeB[(size_t)tx * L + y0 + lane] = strip_gidx(base, L, w);
            edgeA[(size_t)tx * L + y0 + lane] = e3 ? strip_gidx(base, L, e) : -1;
        }
        nact += e3 >> 6;                                 // the east bonds that leave the strip were masked before the count
    }

    if (!FROM_BONDS) {
        nact = __reduce_add_sync(FULLM, nact);
        // satisfied bonds of my 4 columns: Ising counts the unsatisfied ones (2 resp. 4 per bond), Potts the satisfied ones
        uint32_t nsat = (byte_sum(acc_e) >> 1) + (byte_sum(acc_n) >> 2);
        if (ISING) nsat = 8u * (uint32_t)th_eff - nsat;
        uint32_t nminus = byte_sum(acc_m) >> 1;
        if (!colv) nsat = nminus = 0;                    // lanes beyond a ragged edge count nothing
        nsat = __reduce_add_sync(FULLM, nsat);
        if (ISING) nminus = __reduce_add_sync(FULLM, nminus);
        if (lane == 0) {
            AccPart* const part = &acc->part[(tx + 5 * ty) & (ACC_PARTS - 1)];
            if (nact) atomicAdd(&part->n_active, (unsigned long long)nact);
            if (nsat) atomicAdd(&part->sat, (unsigned long long)nsat);
            if (ISING && nminus) atomicAdd(&part->minus, (unsigned long long)nminus);
        }
    }
}
}  // namespace swb
