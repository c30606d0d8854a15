// scan_kernel.cuh -- k_scan: bond activation (P:53 step 1, Eq. 7) fused with strip-local labelling.
// Included by label_kernels.cuh (uses its forest helpers nm_find / nm_root4 / unite_batch and the `prov` encoding).
//
// One warp per TW x TH strip, lane -> 4 consecutive columns, rows in sequence.  A "node" is a horizontal run (inside the
// strip) that has no active north bond from the row above; it is named by its first site.  Every other run adopts the
// name carried by its leftmost contact with the row above, so every name is a node.  When a run has further contacts
// whose names differ from the adopted one, the pair of names is queued; queued pairs are united 32 at a time (all lanes
// busy) in the strip's forest.  Names never depend on the forest, so the row loop has no divergent part.
//
// Names are strip-local site indices (< TW*TH = 4096) kept as 16-bit halves, two per register: P01/P23 = names carried
// by the 4 sites of the previous row, l01/l23 = names of this row.  Which name a site takes is a function of 7 bits --
// the lane's 3 inner east bonds and the 4 north bonds from the row above -- so it comes from a 128-entry table of byte
// permutation selectors (PRMT): 4 permutes name the 4 sites, 2 more (selectors from a second table, indexed by the 4
// east bonds and the link from the previous lane) substitute the names of runs that cross lane boundaries.
#pragma once
#include "common.cuh"

namespace swb {

// ---------------------------------------------------------------------------------------------------- tables
// A half h in [0,4) of a register pair (a, b) seen by PRMT: 0 = a.lo, 1 = a.hi, 2 = b.lo, 3 = b.hi.
constexpr uint32_t lut_half(int h) { return (uint32_t)(((2 * h + 1) << 4) | (2 * h)); }
constexpr uint32_t lut_sel(int hlo, int hhi) { return lut_half(hlo) | (lut_half(hhi) << 8); }

struct ScanLut {
    uint32_t a[128][4];    // index: bits 0,2,4 = E0,E1,E2 (east bonds site j -> j+1 of this row), bits 1,3,5,6 = north bonds
                           // from the previous row into sites 0..3 (the bond byte with bit 7 moved to bit 6)
    uint32_t b[128];       // index: bits 0,2,4,6 = E0..E3 (E3 = east bond into the next lane), bit 1 = EL (link from the
                           // previous lane)
};

constexpr ScanLut make_scan_lut()
{
    ScanLut t{};
    for (int i = 0; i < 128; ++i) {
        const bool E0 = i & 1, E1 = i & 4, E2 = i & 16;
        const int np = ((i >> 1) & 1) | (((i >> 3) & 1) << 1) | (((i >> 5) & 1) << 2) | (((i >> 6) & 1) << 3);
        int s[4] = {0, 0, 0, 0};                         // first site of each site's segment (run inside the lane)
        s[1] = E0 ? 0 : 1;
        s[2] = E1 ? s[1] : 2;
        s[3] = E2 ? s[2] : 3;
        int lc[4] = {-1, -1, -1, -1};                    // leftmost contact of the segment, -1: none
        for (int j = 0; j < 4; ++j)
            for (int k = 3; k >= 0; --k)
                if (s[k] == s[j] && ((np >> k) & 1)) lc[j] = k;
        // X = prmt(P01, P23, selX): the contact names that sites 0 and 1 may take
        const uint32_t selX = lut_sel(lc[0] < 0 ? 0 : lc[0], lc[1] < 0 ? 0 : lc[1]);
        // l01 = prmt(X, NEW01, selL01): contact name, else a new node named by the segment's first site
        const uint32_t selL01 = lut_sel(lc[0] < 0 ? 2 : 0, lc[1] < 0 ? 2 + s[1] : 1);
        // W = prmt(P23, NEW23, selW): names of sites 2 / 3 if they start a segment (s == own index)
        const int wlo = s[2] != 2 ? 0 : (lc[2] < 0 ? 2 : lc[2] - 2);
        const int whi = (np & 8) ? 1 : 3;
        const uint32_t selW = lut_sel(wlo, whi);
        // l23 = prmt(W, l01, selL23): a site whose segment starts at 0 or 1 takes l1
        const uint32_t selL23 = lut_sel(s[2] == 2 ? 0 : 3, s[3] == 3 ? 1 : (s[3] == 2 ? 0 : 3));
        // masks of the sites that have a contact: prmt(0x0000FFFF, x, sel) -> 0xFFFF in the halves with a contact
        const uint32_t m01 = lut_sel((np & 1) ? 0 : 1, (np & 2) ? 0 : 1);
        const uint32_t m23 = lut_sel((np & 4) ? 0 : 1, (np & 8) ? 0 : 1);
        int cnt = 0;                                     // active bonds in the pattern
        for (int k = 0; k < 7; ++k) cnt += (i >> k) & 1;
        t.a[i][0] = selX | (selL01 << 16);
        t.a[i][1] = selW | (selL23 << 16);
        t.a[i][2] = m01 | (m23 << 16);
        // bit 0: the suffix segment (site 3's) has a contact; bit 1: the prefix segment (site 0's) has one; top: count
        t.a[i][3] = (lc[3] >= 0 ? 1u : 0u) | (lc[0] >= 0 ? 2u : 0u) | ((uint32_t)cnt << 28);
    }
    for (int i = 0; i < 128; ++i) {
        const bool E0 = i & 1, E1 = i & 4, E2 = i & 16, E3 = i & 64, EL = i & 2;
        int s[4] = {0, 0, 0, 0};
        s[1] = E0 ? 0 : 1;
        s[2] = E1 ? s[1] : 2;
        s[3] = E2 ? s[2] : 3;
        const bool full = E0 && E1 && E2;
        const bool useP = EL && !full, useS = E3 || (full && EL);
        int h[4] = {0, 1, 0, 1};                         // l01' = prmt(l01, RP|RS<<16, .), l23' = prmt(l23, RP|RS<<16, .)
        for (int j = 0; j < 4; ++j) {
            if (useS && s[j] == s[3]) h[j] = 3;          // in the run that leaves the lane to the right: RS
            else if (useP && s[j] == 0) h[j] = 2;        // in the run that enters from the left: RP
        }
        t.b[i] = lut_sel(h[0], h[1]) | (lut_sel(h[2], h[3]) << 16);
    }
    return t;
}

__device__ const ScanLut d_scan_lut = make_scan_lut();

// ---------------------------------------------------------------------------------------------------- helpers
// PRMT reads the 4 selector nibbles of s[15:0] only (every nibble here is < 8: plain byte select); __byte_perm would
// spend an extra instruction masking the selector.
__device__ __forceinline__ uint32_t prmt(uint32_t a, uint32_t b, uint32_t s)
{
    uint32_t d;
    asm("prmt.b32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(s));
    return d;
}

// d <- 2 d + [u >= T] for T != 0: the carry of u + (2^32 - T) shifted into d.  An add with carry-out (ALU pipe) and an
// add with carry-in (ptxas issues it as IMAD.X on the multiply-add pipe): no compare, select or shift.
__device__ __forceinline__ void shift_in_ge(uint32_t& d, uint32_t u, uint32_t negT)
{
    asm("{\n\t.reg .u32 t;\n\tadd.cc.u32 t, %1, %2;\n\taddc.u32 %0, %0, %0;\n\t}" : "+r"(d) : "r"(u), "r"(negT));
}

// Draw byte of the 4 sites whose first pair has Philox counter c0, at step (t_lo, t_hi): bit 2j = [east draw of site j
// >= T], bit 2j+1 = [north draw >= T] (S:8c.3: u(i,d,t) = PHILOX(seed; i>>1, t, BOND)[2(i&1)+d]).  A pure function of
// (seed, t, site, T): k_final computes it one sweep ahead (draw cache, see k_final) and k_scan<SRC_DRAWS> only reads it.
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
__device__ __forceinline__ uint32_t bond_byte(const Params& p, uint32_t d, uint32_t w, uint32_t e, uint32_t n)
{
    uint32_t eq;                                         // bit 8j+1: s_j == s_east, bit 8j+2: s_j == s_north
    if (ISING) {                                         // bytes 0x01 / 0xFF: equal <=> bit 1 (and bit 2) of the xor is 0
        eq = (~(w ^ e) & 0x02020202u) | (~(w ^ n) & 0x04040404u);
    } else {
        eq = (__vcmpeq4(w, e) & 0x02020202u) | (__vcmpeq4(w, n) & 0x04040404u);
    }
    // gather the 4 bit pairs (8j+1, 8j+2) into bits (2j, 2j+1) of the high word; the cross terms of the product land on
    // distinct bits below 32 or above bit 7 of the high word (no carries)
    // p.dmask = 0xFF, or 0 if T = 0 (then u >= T always, but u + 2^32 never carries)
    return __umulhi(eq, 0x82082000u) & ~d & p.dmask;     // 2^31 + 2^25 + 2^19 + 2^13
}

// Draw cache (workspace): one 32-bit word per lane and group of 4 rows of a strip, byte r = draw byte of row 4g + r:
// word index ((ty * ntx + tx) * (TH / 4) + g) * 32 + lane.  Written by k_final<MODE_SW> for step t+1 (its warp g owns rows
// 4g..4g+3), read by k_scan<SRC_DRAWS> of the next sweep.
__device__ __forceinline__ size_t draw_word_index(const Params& p, int tx, int ty, int g, int lane)
{
    return ((size_t)(ty * p.ntx + tx) * (TH / 4) + g) * 32 + lane;
}

// ---------------------------------------------------------------------------------------------------- k_scan
// SRC_PHILOX: read spins, draw bonds (a1).  SRC_DRAWS: read spins and the draw cache k_final filled one sweep ahead (the
// same bonds, the Philox work done where the issue slots were idle).  SRC_BONDS: read packed bonds (sw_label).  Writes the
// provisional labels (`prov`, see label_kernels.cuh) and the edge arrays, and adds the number of active bonds to
// acc->n_active.  FULLW: L is a multiple of TW, every strip has all 32 lanes (no ragged right edge; the predicates fold away).
enum { SRC_PHILOX = 0, SRC_BONDS = 1, SRC_DRAWS = 2 };
template <int SRC, bool ISING, bool FULLW>
__global__ void __launch_bounds__(SCAN_THREADS)
k_scan(const Params p, const uint32_t* __restrict__ spins_w, const uint8_t* __restrict__ bonds_in,
       const uint32_t* __restrict__ draws, int* prov, int* __restrict__ edgeA, int* __restrict__ edgeB,
       Acc* __restrict__ acc)
{
    constexpr bool FROM_BONDS = SRC == SRC_BONDS;
    __shared__ __align__(16) uint16_t s_nm[SCAN_WARPS][TW * TH];
    __shared__ uint32_t s_q[SCAN_WARPS][QCAP];
    __shared__ __align__(16) uint4 s_la[128];
    __shared__ uint32_t s_lb[128];
    for (int i = threadIdx.x; i < 128; i += SCAN_THREADS)
        s_la[i] = make_uint4(d_scan_lut.a[i][0], d_scan_lut.a[i][1], d_scan_lut.a[i][2], d_scan_lut.a[i][3]);
    for (int i = threadIdx.x; i < 128; i += SCAN_THREADS) s_lb[i] = d_scan_lut.b[i];
    __syncthreads();                                     // the only block-wide barrier

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int tx = blockIdx.x * SCAN_WARPS + warp, ty = blockIdx.y;
    if (tx >= p.ntx) return;
    uint16_t* nm = s_nm[warp];
    volatile uint16_t* vnm = nm;
    volatile uint32_t* q = s_q[warp];
    const int L = p.L, Lw = L >> 2;
    const int x0 = tx * TW, y0 = ty * TH;
    const int tw_eff = FULLW ? TW : min(TW, L - x0), th_eff = FULLW ? TH : min(TH, L - y0);   // TH divides TW
    const int x = x0 + 4 * lane;
    const bool colv = FULLW || 4 * lane < tw_eff;
    const int last_lane = (tw_eff >> 2) - 1;             // lane that owns the strip's last column
    const bool is_last = lane == last_lane;
    const int base = y0 * L + x0;
    const int xw = x >> 2;
    const int xew = ((x + 4 == L) ? 0 : x + 4) >> 2;     // east halo word of the last lane (periodic)
    const unsigned lt = lanemask_lt(), me = 1u << lane, le = lt | me, gt = ~le;
    // the east bond that leaves the strip is dropped from the lane's bond byte; lanes beyond a ragged edge have no bonds
    const uint32_t gmask = !colv ? 0u : is_last ? 0xBFu : 0xFFu;

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
    uint32_t npm = 0;                                    // north bonds from the previous row into this row (bits 1,3,5,6)
    uint32_t NEW01 = (uint32_t)(4 * lane) * 0x00010001u + 0x00010000u;      // own names of sites 0,1 / 2,3 of this row
    uint32_t NEW23 = NEW01 + 0x00020002u;
    uint32_t nact = 0;
    int qn = 0;                                          // queued pairs (warp-uniform)
    uint32_t eastm = 0;                                  // bit (th_eff-1-ly) = the east bond of site 3 in row ly (last lane: it leaves the strip)
    uint32_t northm = 0;                                 // bond byte of the last row: its north bonds (bits 1,3,5,7) leave the strip

    // running per-row quantities: Philox counter of the lane's first pair, global index of the lane's first site, pointer
    // to the lane's spin word of the row to prefetch (ly + 3)
    uint32_t c0 = (uint32_t)(y0 * L + x) >> 1;
    int gi = y0 * L + x;
    const uint32_t* pw = spins_w + (size_t)(y0 + 3) * Lw + xws;   // the lane's word of the row to prefetch; halo: + dxe
    const uint32_t* const pw_halo = spins_w + row_halo + xws;
    const int dxe = xew - xws;

    uint32_t dw = 0;                                     // draw bytes of the rows 4g..4g+3 (SRC_DRAWS)
    const uint32_t* pdw = draws + (SRC == SRC_DRAWS ? draw_word_index(p, tx, ty, 0, lane) : 0);
    for (int ly = 0; ly < th_eff; ++ly) {
        uint32_t G = 0;                                  // the lane's bond byte of this row
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
            G = bond_byte<ISING>(p, d, w0, east, w1);
            c0 += (uint32_t)L >> 1;
            w0 = w1; w1 = w2; w2 = w3; h0 = h1; h1 = h2; h2 = h3;
        } else if (colv) {
            G = bonds_in[(size_t)gi >> 2];
        }
        // bonds that leave the strip are remembered for the edge arrays and dropped here
        // (the north bonds of the last row are not used inside the loop: they only feed the next row's table index)
        eastm = eastm * 2u + ((G >> 6) & 1u);
        G &= gmask;
        northm = G;

        // ---- names of this row's sites ----------------------------------------------------------------------
        const uint32_t EL = (__shfl_up_sync(FULLM, G, 1) >> 5) & (lane ? 2u : 0u);
        const uint4 A = s_la[(G & 0x15u) | npm];
        const uint32_t Bf = s_lb[(G & 0x55u) | EL];
        const uint32_t X = prmt(P01, P23, A.x);
        uint32_t l01 = prmt(X, NEW01, A.x >> 16);
        const uint32_t W = prmt(P23, NEW23, A.y);
        uint32_t l23 = prmt(W, l01, A.y >> 16);
        nact += A.w >> 28;

        // runs that cross lane boundaries: lanes a..b, a's suffix segment, full lanes, b's prefix segment
        const bool E3 = G & 0x40u;
        const unsigned LINK = __ballot_sync(FULLM, E3);
        const unsigned FULLB = __ballot_sync(FULLM, (G & 0x15u) == 0x15u);
        const unsigned CS = __ballot_sync(FULLM, (A.w & 1u) != 0u);
        const unsigned CP = __ballot_sync(FULLM, (A.w & 2u) != 0u);
        const unsigned nPTL = ~(FULLB & (LINK << 1));                       // lanes where a run cannot pass to the left
        const unsigned nPTR = ~(FULLB & LINK);                              // ... to the right
        const int a_le = 31 - __clz(nPTL & le);                             // bit 0 of nPTL is always set
        const int bS = E3 ? __ffs(nPTR & gt) - 1 : lane;                    // bit 31 of nPTR is always set
        const unsigned MS = (CS & ((1u << bS) - 1u) & (FULLM << a_le)) | (CP & (1u << bS));
        const int srcS = MS ? __ffs(MS) - 1 : a_le;                         // lane that holds the run's name
        const uint32_t pub = prmt(l01, l23, 0x7610);                        // l0 | l3 << 16
        const uint32_t v = __shfl_sync(FULLM, pub, srcS);
        const uint32_t RS = prmt(v, 0u, srcS == bS ? 0x4410u : 0x4432u);    // the last lane's prefix name, else a suffix name
        const uint32_t RPS = prmt(__shfl_up_sync(FULLM, RS, 1), RS, 0x5410);   // RP | RS << 16
        l01 = prmt(l01, RPS, Bf);
        l23 = prmt(l23, RPS, Bf >> 16);

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

        // contacts whose carried name differs from the adopted one: queue the pair of names
        {
            const uint32_t d01 = (P01 ^ l01) & prmt(0x0000FFFFu, 0u, A.z);
            const uint32_t d23 = (P23 ^ l23) & prmt(0x0000FFFFu, 0u, A.z >> 16);
            const bool m0 = d01 & 0xFFFFu, m1 = d01 >> 16, m2 = d23 & 0xFFFFu, m3 = d23 >> 16;
            const unsigned B0 = __ballot_sync(FULLM, m0), B1 = __ballot_sync(FULLM, m1);
            const unsigned B2 = __ballot_sync(FULLM, m2), B3 = __ballot_sync(FULLM, m3);
            volatile uint32_t* qp = q + qn;
            if (m0) qp[__popc(B0 & lt)] = prmt(l01, P01, 0x5410);
            qp += __popc(B0);
            if (m1) qp[__popc(B1 & lt)] = prmt(l01, P01, 0x7632);
            qp += __popc(B1);
            if (m2) qp[__popc(B2 & lt)] = prmt(l23, P23, 0x5410);
            qp += __popc(B2);
            if (m3) qp[__popc(B3 & lt)] = prmt(l23, P23, 0x7632);
            qp += __popc(B3);
            qn = (int)(qp - q);
        }
        if (qn >= 32) {
            __syncwarp();                                // queue, forest entries and `prov` rows visible to the whole warp
            do {
                qn -= 32;
                unite_batch(vnm, true, q[qn + lane], prov, base, L);
            } while (qn >= 32);
            __syncwarp();                                // queue slots read before the next row overwrites them
        }

        P01 = l01; P23 = l23;
        npm = (G & 0x2Au) | ((G >> 1) & 0x40u);
        NEW01 += (uint32_t)TW * 0x00010001u;
        NEW23 += (uint32_t)TW * 0x00010001u;
        gi += L;
    }

    northm &= 0xAAu;
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
            n.x = (northm & 0x02u) ? strip_gidx(base, L, n0) : -1;
            n.y = (northm & 0x08u) ? strip_gidx(base, L, n1) : -1;
            n.z = (northm & 0x20u) ? strip_gidx(base, L, n2) : -1;
            n.w = (northm & 0x80u) ? strip_gidx(base, L, n3) : -1;
            *reinterpret_cast<int4*>(edgeB + (size_t)nE + (size_t)ty * L + x) = s;
            *reinterpret_cast<int4*>(edgeA + (size_t)nE + (size_t)ty * L + x) = n;
        }
        // first column -> rootW, last column -> rootE: lane i takes row i
        const uint32_t em = __shfl_sync(FULLM, eastm, last_lane);           // row ly at bit th_eff-1-ly
        if (lane < th_eff) {
            int w = lane * TW, e = lane * TW + tw_eff - 1, w2 = w, e2 = e;
            nm_root4(vnm, w, e, w2, e2);
            edgeB[(size_t)tx * L + y0 + lane] = strip_gidx(base, L, w);
            edgeA[(size_t)tx * L + y0 + lane] = ((em >> (th_eff - 1 - lane)) & 1u) ? strip_gidx(base, L, e) : -1;
        }
    }

    if (!FROM_BONDS) {
        nact += __popc(northm);
        if (colv) nact += __popc(eastm);                 // my east bonds into the next lane / out of the strip, all rows
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) nact += __shfl_xor_sync(FULLM, nact, o);
        if (lane == 0 && nact)
            atomicAdd(&acc->part[(tx + 5 * ty) & (ACC_PARTS - 1)].n_active, (unsigned long long)nact);
    }
}

}  // namespace swb
