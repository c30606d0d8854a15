/*
 * sw_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, serial, obviously-correct CPU statement of the Swendsen-Wang cluster
 * update of the 2D q-state Potts / Ising model on a periodic L x L square
 * lattice (M. Weigel, arXiv:1105.5804; citations "P:NN" are line numbers of
 * /root/reference/PAPER.md, "S:8c.n" are definitions n of SURVEY.md section
 * 8(c), the reading of the paper this repository builds to).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may call this.  It shares no code with the CUDA path
 * under paper_1105_5804_b200/csrc (it has its own Philox, its own index maps,
 * its own labelling).  Integer arithmetic only, except the threshold, which is
 * IEEE double as the paper's p = 1 - exp(-beta J).
 *
 * What pins each function (tests/test_oracle_*.py, all `-m "not gpu"`):
 *   orc_philox4x32_10   Random123 known-answer vectors (tests/golden/philox_kat.txt)
 *   orc_threshold       closed forms (p_c = 2 - sqrt 2, p = 2/3, p = 1/2, ...)
 *   orc_bonds           T=0 / T=max special cases, never joins unequal spins,
 *                       mean bond density = p * sat / 2N within binomial error
 *   orc_label           all 2^18 bond configurations of the 3x3 torus against
 *                       an independent transitive closure; special patterns;
 *                       invariants (canonical minimum, sizes sum to N)
 *   orc_flip / orc_sweep / orc_run_chain
 *                       exact enumeration of the 4x4 Ising model (<E>, <|m|>,
 *                       <m^2>, energy histogram chi^2), Kaufman's exact
 *                       finite-L energy at L=64, FK identity <sum size^2> = N^2 <m^2>,
 *                       q=4 L=4 transfer-matrix energy, survey golden vectors
 *   orc_wolff_step      equals "label everything, flip the seed's cluster";
 *                       4x4 exact <E>, <|m|>; survey golden vectors
 *   orc_observables     brute-force E and M in the test, closed forms for
 *                       cold / checkerboard / stripe configurations
 *   orc_cluster_stats   numpy bincount on the same labels; percolation
 *                       p=1/2 cluster density, Euler duality n(0.3)-n(0.7)=0.4
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <math.h>

/* ---- Philox4x32-10 (S:8c preamble; Salmon et al., SC'11; the paper's own RNG
 * was a per-thread LCG, replaced because its stream depends on the
 * thread layout) ------------------------------------------------------------ */
#define PHILOX_M0 0xD2511F53u
#define PHILOX_M1 0xCD9E8D57u
#define PHILOX_W0 0x9E3779B9u
#define PHILOX_W1 0xBB67AE85u

void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)PHILOX_M0 * (uint64_t)c0;
        uint64_t p1 = (uint64_t)PHILOX_M1 * (uint64_t)c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += PHILOX_W0;
        k1 += PHILOX_W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* S:8c.2 -- counter word c3 selects the domain; (c1,c2) = step counter t. */
enum { DOM_INIT = 0, DOM_BOND = 1, DOM_FLIP = 2, DOM_WSEED = 3 };

static void draw(uint64_t seed, uint32_t c0, uint64_t t, uint32_t dom, uint32_t w[4])
{
    uint32_t ctr[4] = { c0, (uint32_t)(t & 0xFFFFFFFFu), (uint32_t)(t >> 32), dom };
    uint32_t key[2] = { (uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32) };
    orc_philox4x32_10(ctr, key, w);
}

/* uniform integer in [0,n) from 32 random bits: multiply-high (S:8c issue 10) */
static uint32_t mulhi_range(uint32_t w, uint32_t n)
{
    return (uint32_t)(((uint64_t)w * (uint64_t)n) >> 32);
}

/* ---- threshold: p = 1 - exp(-K beta), K = 2 for the Ising +-1 convention
 * (q=2), K = 1 for the Potts delta convention (P:45 Eq. below (4); S:8c.4) ---- */
uint32_t orc_threshold(int q, double beta)
{
    double K = (q == 2) ? 2.0 : 1.0;
    double p = 1.0 - exp(-K * beta);
    double v = floor(p * 4294967296.0);
    if (v < 0.0) v = 0.0;
    if (v > 4294967295.0) v = 4294967295.0;
    return (uint32_t)v;
}

uint32_t orc_threshold_from_p(double p)
{
    double v = floor(p * 4294967296.0);
    if (v < 0.0) v = 0.0;
    if (v > 4294967295.0) v = 4294967295.0;
    return (uint32_t)v;
}

/* ---- index maps (S:8c.1; P:66 periodic square lattice; Fig. 1 P:86-96:
 * site 0 bottom-left, i = y L + x) ------------------------------------------ */
static int64_t east_of(int64_t L, int64_t i)  { int64_t x = i % L, y = i / L; return y * L + (x + 1) % L; }
static int64_t north_of(int64_t L, int64_t i) { int64_t x = i % L, y = i / L; return ((y + 1) % L) * L + x; }
static int64_t west_of(int64_t L, int64_t i)  { int64_t x = i % L, y = i / L; return y * L + (x + L - 1) % L; }
static int64_t south_of(int64_t L, int64_t i) { int64_t x = i % L, y = i / L; return ((y + L - 1) % L) * L + x; }

/* stored byte <-> Potts state k in [0,q): q=2 stores s=+1 for k=0, s=-1 for k=1
 * (Ising convention); q>2 stores k itself (S:8b conventions). */
static int8_t store_of(int q, uint32_t k) { return (q == 2) ? (int8_t)(k ? -1 : 1) : (int8_t)k; }

/* ---- S:8c.8 initialisation --------------------------------------------------- */
int orc_init_spins(int32_t L, int32_t q, uint64_t seed, int32_t mode, int8_t *spins)
{
    int64_t N = (int64_t)L * L;
    if (L < 3 || q < 2 || q > 8) return -1;
    for (int64_t i = 0; i < N; ++i) {
        uint32_t k = 0;
        if (mode == 1) {
            uint32_t w[4];
            draw(seed, (uint32_t)(i >> 2), 0, DOM_INIT, w);
            k = mulhi_range(w[i & 3], (uint32_t)q);
        }
        spins[i] = store_of(q, k);
    }
    return 0;
}

/* ---- S:8c.3 + 8c.4 bond activation (P:53 step 1; Eq. 7):
 *   n(i,d) = [s_i == s_nbr(i,d)] and [u(i,d,t) < T],
 *   u(i,d,t) = PHILOX(seed; i>>1, t_lo, t_hi, BOND)[2 (i&1) + d], d=0 east, d=1 north.
 * Output: one byte per site, bit0 = east bond, bit1 = north bond.  Returns the
 * number of active bonds. */
int64_t orc_bonds(int32_t L, uint32_t T, uint64_t seed, uint64_t t,
                  const int8_t *spins, uint8_t *codes)
{
    int64_t N = (int64_t)L * L, active = 0;
    for (int64_t i = 0; i < N; ++i) {
        uint32_t w[4];
        draw(seed, (uint32_t)(i >> 1), t, DOM_BOND, w);
        uint32_t ue = w[2 * (i & 1) + 0];
        uint32_t un = w[2 * (i & 1) + 1];
        int e = (spins[i] == spins[east_of(L, i)])  && (ue < T);
        int n = (spins[i] == spins[north_of(L, i)]) && (un < T);
        codes[i] = (uint8_t)(e | (n << 1));
        active += e + n;
    }
    return active;
}

/* packed form used at the C-ABI boundary (S:8b): byte b holds sites 4b..4b+3,
 * site j uses bits 2(j&3) (east) and 2(j&3)+1 (north). */
void orc_pack_bonds(int64_t N, const uint8_t *codes, uint8_t *packed)
{
    for (int64_t b = 0; b < (N + 3) / 4; ++b) packed[b] = 0;
    for (int64_t i = 0; i < N; ++i)
        packed[i >> 2] |= (uint8_t)((codes[i] & 3u) << (2 * (i & 3)));
}

void orc_unpack_bonds(int64_t N, const uint8_t *packed, uint8_t *codes)
{
    for (int64_t i = 0; i < N; ++i)
        codes[i] = (uint8_t)((packed[i >> 2] >> (2 * (i & 3))) & 3u);
}

/* ---- S:8c.5 labelling by breadth-first search (section II.B.1): seeds in
 * increasing order, FIFO queue, every reached site gets the seed's index, hence
 * label = minimum site index of the component.  Returns the cluster count. */
int64_t orc_label(int32_t L, const uint8_t *codes, int32_t *labels)
{
    int64_t N = (int64_t)L * L, nclusters = 0;
    int32_t *queue = (int32_t *)malloc((size_t)N * sizeof(int32_t));
    if (!queue) return -1;
    for (int64_t i = 0; i < N; ++i) labels[i] = -1;
    for (int64_t seed_site = 0; seed_site < N; ++seed_site) {
        if (labels[seed_site] != -1) continue;
        ++nclusters;
        int64_t head = 0, tail = 0;
        labels[seed_site] = (int32_t)seed_site;
        queue[tail++] = (int32_t)seed_site;
        while (head < tail) {
            int64_t i = queue[head++];
            int64_t nb;
            if (codes[i] & 1) {                              /* my east bond  */
                nb = east_of(L, i);
                if (labels[nb] == -1) { labels[nb] = (int32_t)seed_site; queue[tail++] = (int32_t)nb; }
            }
            if (codes[i] & 2) {                              /* my north bond */
                nb = north_of(L, i);
                if (labels[nb] == -1) { labels[nb] = (int32_t)seed_site; queue[tail++] = (int32_t)nb; }
            }
            nb = west_of(L, i);
            if (codes[nb] & 1) {                             /* west neighbour's east bond */
                if (labels[nb] == -1) { labels[nb] = (int32_t)seed_site; queue[tail++] = (int32_t)nb; }
            }
            nb = south_of(L, i);
            if (codes[nb] & 2) {                             /* south neighbour's north bond */
                if (labels[nb] == -1) { labels[nb] = (int32_t)seed_site; queue[tail++] = (int32_t)nb; }
            }
        }
    }
    free(queue);
    return nclusters;
}

/* ---- S:8c.6 flip (P:55 step 3): new state of cluster r is
 *   k_r = (PHILOX(seed; r, t_lo, t_hi, FLIP)[0] * q) >> 32, every site takes k_{label}. */
void orc_flip(int32_t L, int32_t q, uint64_t seed, uint64_t t,
              const int32_t *labels, int8_t *spins)
{
    int64_t N = (int64_t)L * L;
    for (int64_t i = 0; i < N; ++i) {
        uint32_t w[4];
        draw(seed, (uint32_t)labels[i], t, DOM_FLIP, w);
        spins[i] = store_of(q, mulhi_range(w[0], (uint32_t)q));
    }
}

/* ---- S:8c.7 / S:8a a6 observables (Eq. 1), int64 ------------------------- */
typedef struct {
    int64_t sat_bonds;       /* # bonds (of 2N) whose end spins are equal        */
    int64_t energy;          /* Ising: -(2 sat - 2N) = -sum s_i s_j; Potts: -sat */
    int64_t magnetisation;   /* Ising: sum s_i; Potts: q max_k n_k - N           */
    int64_t state_count[8];  /* n_k                                              */
} orc_obs;

void orc_observables(int32_t L, int32_t q, const int8_t *spins, orc_obs *o)
{
    int64_t N = (int64_t)L * L;
    memset(o, 0, sizeof(*o));
    for (int64_t i = 0; i < N; ++i) {
        o->sat_bonds += (spins[i] == spins[east_of(L, i)]);
        o->sat_bonds += (spins[i] == spins[north_of(L, i)]);
        int k = (q == 2) ? (spins[i] == 1 ? 0 : 1) : (int)(uint8_t)spins[i];
        if (k >= 0 && k < 8) o->state_count[k] += 1;
    }
    if (q == 2) {
        o->energy = -(2 * o->sat_bonds - 2 * N);
        o->magnetisation = o->state_count[0] - o->state_count[1];
    } else {
        int64_t mx = 0;
        for (int k = 0; k < q; ++k) if (o->state_count[k] > mx) mx = o->state_count[k];
        o->energy = -o->sat_bonds;
        o->magnetisation = (int64_t)q * mx - N;
    }
}

/* ---- S:8a a9 cluster statistics from canonical labels -------------------------- */
typedef struct {
    int64_t  n_clusters;
    int64_t  max_cluster;
    uint64_t sum_sq_cluster;
    int64_t  hist32[32];     /* bin b counts clusters with 2^b <= size < 2^(b+1) */
} orc_cstats;

int orc_cluster_stats(int64_t N, const int32_t *labels, orc_cstats *c)
{
    int32_t *size = (int32_t *)calloc((size_t)N, sizeof(int32_t));
    if (!size) return -1;
    memset(c, 0, sizeof(*c));
    for (int64_t i = 0; i < N; ++i) size[labels[i]] += 1;
    for (int64_t i = 0; i < N; ++i) {
        if (labels[i] != i) continue;
        int64_t s = size[i];
        c->n_clusters += 1;
        if (s > c->max_cluster) c->max_cluster = s;
        c->sum_sq_cluster += (uint64_t)s * (uint64_t)s;
        int b = 0;
        while ((s >> (b + 1)) != 0) ++b;
        c->hist32[b] += 1;
    }
    free(size);
    return 0;
}

/* ---- one full SW sweep (P:51-55 steps 1-3) at step counter t.  Optional
 * outputs may be NULL.  Returns the cluster count; *active gets the bond count. */
int64_t orc_sweep(int32_t L, int32_t q, uint32_t T, uint64_t seed, uint64_t t,
                  int8_t *spins, int32_t *labels, uint8_t *codes, int64_t *active)
{
    int64_t N = (int64_t)L * L;
    int own_labels = (labels == NULL), own_codes = (codes == NULL);
    if (own_labels) labels = (int32_t *)malloc((size_t)N * sizeof(int32_t));
    if (own_codes)  codes  = (uint8_t *)malloc((size_t)N);
    if (!labels || !codes) return -1;
    int64_t nb = orc_bonds(L, T, seed, t, spins, codes);
    int64_t nc = orc_label(L, codes, labels);
    orc_flip(L, q, seed, t, labels, spins);
    if (active) *active = nb;
    if (own_labels) free(labels);
    if (own_codes)  free(codes);
    return nc;
}

/* ---- a chain of n sweeps starting at counter t0, recording after every sweep:
 * series[4*s + 0..3] = energy, magnetisation, n_clusters, sum of squared
 * cluster sizes (of the labelling inside that sweep).  Used by the statistical
 * pins so that 10^6 sweeps of a 4x4 lattice do not pay a Python call each. */
int orc_run_chain(int32_t L, int32_t q, uint32_t T, uint64_t seed, uint64_t t0,
                  int64_t n, int8_t *spins, int64_t *series)
{
    int64_t N = (int64_t)L * L;
    int32_t *labels = (int32_t *)malloc((size_t)N * sizeof(int32_t));
    uint8_t *codes = (uint8_t *)malloc((size_t)N);
    if (!labels || !codes) return -1;
    for (int64_t s = 0; s < n; ++s) {
        int64_t nb = 0;
        int64_t nc = orc_sweep(L, q, T, seed, t0 + (uint64_t)s, spins, labels, codes, &nb);
        if (series) {
            orc_obs o; orc_cstats c;
            orc_observables(L, q, spins, &o);
            orc_cluster_stats(N, labels, &c);
            series[4 * s + 0] = o.energy;
            series[4 * s + 1] = o.magnetisation;
            series[4 * s + 2] = nc;
            series[4 * s + 3] = (int64_t)c.sum_sq_cluster;
        }
    }
    free(labels); free(codes);
    return 0;
}

/* ---- S:8c.9 Wolff single-cluster step: seed site from Philox, grow the
 * cluster by BFS over the bonds of step t evaluated on the PRE-step spins
 * (bond draws are pure functions of (seed,t,site,direction), so this equals
 * "SW-decompose, pick a site, flip its cluster", P:330/P:334 option (a)), then
 * flip it (Ising: s -> -s).  Returns |C|; *seed_site / *root get the seed site and
 * the minimum site index of the cluster.  q must be 2 (S:8c issue 8). */
int64_t orc_wolff_step(int32_t L, int32_t q, uint32_t T, uint64_t seed, uint64_t t,
                       int8_t *spins, int64_t *seed_site, int64_t *root)
{
    int64_t N = (int64_t)L * L;
    if (q != 2) return -1;
    uint32_t w[4];
    draw(seed, 0u, t, DOM_WSEED, w);
    int64_t i0 = (int64_t)(((uint64_t)w[0] * (uint64_t)N) >> 32);
    uint8_t *visited = (uint8_t *)calloc((size_t)N, 1);
    int32_t *queue = (int32_t *)malloc((size_t)N * sizeof(int32_t));
    if (!visited || !queue) return -1;
    int8_t s0 = spins[i0];
    int64_t head = 0, tail = 0, minidx = i0;
    visited[i0] = 1; queue[tail++] = (int32_t)i0;
    while (head < tail) {
        int64_t i = queue[head++];
        if (i < minidx) minidx = i;
        /* the four bonds of site i; bond (i,east) belongs to i, bond (west,east) to west, ... */
        int64_t nbr[4]   = { east_of(L, i), north_of(L, i), west_of(L, i), south_of(L, i) };
        int64_t owner[4] = { i, i, nbr[2], nbr[3] };
        int     dir[4]   = { 0, 1, 0, 1 };
        for (int b = 0; b < 4; ++b) {
            int64_t j = nbr[b];
            if (visited[j] || spins[j] != s0) continue;   /* unvisited sites still carry pre-step spins */
            uint32_t u[4];
            draw(seed, (uint32_t)(owner[b] >> 1), t, DOM_BOND, u);
            if (u[2 * (owner[b] & 1) + dir[b]] < T) { visited[j] = 1; queue[tail++] = (int32_t)j; }
        }
    }
    for (int64_t k = 0; k < tail; ++k) spins[queue[k]] = (int8_t)(-s0);
    if (seed_site) *seed_site = i0;
    if (root) *root = minidx;
    free(visited); free(queue);
    return tail;
}

/* chain of n Wolff steps; series[3*s + 0..2] = energy, magnetisation, |C| */
int orc_wolff_chain(int32_t L, uint32_t T, uint64_t seed, uint64_t t0, int64_t n,
                    int8_t *spins, int64_t *series)
{
    for (int64_t s = 0; s < n; ++s) {
        int64_t sz = orc_wolff_step(L, 2, T, seed, t0 + (uint64_t)s, spins, NULL, NULL);
        if (sz < 0) return -1;
        if (series) {
            orc_obs o;
            orc_observables(L, 2, spins, &o);
            series[3 * s + 0] = o.energy;
            series[3 * s + 1] = o.magnetisation;
            series[3 * s + 2] = sz;
        }
    }
    return 0;
}

/* FNV-1a 64-bit of a byte buffer (golden-vector fingerprints, S:8c last table) */
uint64_t orc_fnv1a64(const uint8_t *p, int64_t n)
{
    uint64_t h = 0xcbf29ce484222325ull;
    for (int64_t i = 0; i < n; ++i) { h ^= p[i]; h *= 0x100000001b3ull; }
    return h;
}

/* ---- S:8f row 1, second half: the few-cluster variant.  The paper grows clusters from
 * several seed sites at once and gives every cluster "a flipping probability p_flip < 1"; it states that this is
 * "logically identical to performing the full SW decomposition and then selecting [...] points on the lattice,
 * followed by flipping all distinct clusters these points belong to".  That statement is what is written out here
 * (reading 21 fixes what the paper leaves open -- the draws):
 *   bonds and labels of step t as in a sweep (S:8c.3-5, on the pre-step spins);
 *   seed sites i_k = (PHILOX(seed; k, t, WSEED)[0] * N) >> 32, k = 0 .. n_seeds-1 (k = 0 is the Wolff seed, S:8c.9);
 *   a cluster is selected iff it holds at least one seed site (a cluster hit twice is one cluster);
 *   a selected cluster with root r is flipped (s -> -s on all its sites) iff PHILOX(seed; r, t, FLIP)[1] < T_flip
 *   (word 1: word 0 is the state draw of a sweep), T_flip = floor(p_flip 2^32), so p_flip < 1 always.
 * Returns the number of flipped sites; *n_flipped_clusters the number of flipped clusters; labels_out (N, or
 * NULL) the canonical labels of the decomposition.  q must be 2 (as for Wolff).  t += 1 is the caller's.
 * Pins (tests/test_oracle_physics.py): a numpy restatement from the pinned bonds / labels / Philox; one seed at
 * T_flip = 2^32 - 1 equals orc_wolff_step (ties the seed keying to the golden Wolff vectors); exact <E>, <|m|> of
 * the 4 x 4 Ising model for a chain with 3 seeds and p_flip = 0.7 (detailed balance holds cluster by cluster). */
int64_t orc_fewcluster_step(int32_t L, int32_t q, uint32_t T, uint64_t seed, uint64_t t, int32_t n_seeds,
                            uint32_t T_flip, int8_t *spins, int32_t *labels_out, int64_t *n_flipped_clusters)
{
    int64_t N = (int64_t)L * L, flipped = 0, nfc = 0;
    if (q != 2 || n_seeds < 0) return -1;
    uint8_t *codes = (uint8_t *)malloc((size_t)N);
    int32_t *labels = (int32_t *)malloc((size_t)N * sizeof(int32_t));
    uint8_t *selected = (uint8_t *)calloc((size_t)N, 1);          /* selected[r]: root r holds a seed site */
    if (!codes || !labels || !selected) { free(codes); free(labels); free(selected); return -1; }
    orc_bonds(L, T, seed, t, spins, codes);
    orc_label(L, codes, labels);
    for (int32_t k = 0; k < n_seeds; ++k) {
        uint32_t w[4];
        draw(seed, (uint32_t)k, t, DOM_WSEED, w);
        int64_t ik = (int64_t)(((uint64_t)w[0] * (uint64_t)N) >> 32);
        selected[labels[ik]] = 1;
    }
    for (int64_t i = 0; i < N; ++i) {
        int32_t r = labels[i];
        if (!selected[r]) continue;
        uint32_t w[4];
        draw(seed, (uint32_t)r, t, DOM_FLIP, w);
        if (w[1] < T_flip) {
            spins[i] = (int8_t)(-spins[i]);
            ++flipped;
            if (i == r) ++nfc;
        }
    }
    if (labels_out) memcpy(labels_out, labels, (size_t)N * sizeof(int32_t));
    if (n_flipped_clusters) *n_flipped_clusters = nfc;
    free(codes); free(labels); free(selected);
    return flipped;
}

/* chain of n few-cluster steps; series[3*s + 0..2] = energy, magnetisation, flipped sites */
int orc_fewcluster_chain(int32_t L, uint32_t T, uint64_t seed, uint64_t t0, int64_t n, int32_t n_seeds,
                         uint32_t T_flip, int8_t *spins, int64_t *series)
{
    for (int64_t s = 0; s < n; ++s) {
        int64_t f = orc_fewcluster_step(L, 2, T, seed, t0 + (uint64_t)s, n_seeds, T_flip, spins, NULL, NULL);
        if (f < 0) return -1;
        if (series) {
            orc_obs o;
            orc_observables(L, 2, spins, &o);
            series[3 * s + 0] = o.energy;
            series[3 * s + 1] = o.magnetisation;
            series[3 * s + 2] = f;
        }
    }
    return 0;
}

/* ==================================================================================
 * Simple cubic lattice ("hypercubic lattices", P:154
 * "three out of six neighbours" are looked after by every site in 3D).  The same
 * three steps on a periodic L x L x L lattice, site i = z L^2 + y L + x,
 * each site owning its bonds to the east (x+1), north (y+1) and up (z+1) neighbour.
 * DESIGN.md reading 19 (the survey fixes the draws for two directions only):
 *   u3(i,d,t) = PHILOX(seed; i, t_lo, t_hi, BOND3)[d],  d = 0 east, 1 north, 2 up,
 * one call per site, word 3 unused, domain BOND3 = 4.  Initialisation, threshold and
 * flip are the 2D definitions over N = L^3 sites (S:8c.4, 8c.6, 8c.8).
 *
 * Pins (tests/test_oracle_cubic.py): orc3_bonds -- T = 0 / T = max, never joins
 * unequal spins, the three directions hit the three distinct neighbours (single-spin
 * patterns), density; orc3_label -- random bond sets on 3^3 .. 6^3 against an
 * independent transitive closure and scipy's connected components, wrap bonds in all
 * three directions; orc3_observables -- numpy definition, closed forms (cold, layered);
 * orc3_sweep / orc3_run_chain -- exact <E>, <|m|>, <m^2> of the 3 x 3 x 3 Ising model
 * (sum over all 2^27 states, done plane by plane in the test) and the FK identity;
 * orc3_init_spins -- equals orc_init_spins at equal N (golden L4_init_k pins that one)
 * and the keying (i>>2, 0, 0, INIT)[i&3] rebuilt from the KAT-pinned Philox;
 * orc3_flip -- constant on clusters, k_r rebuilt per root from the pinned Philox with
 * both words of t in use, Ising storage (a slipped counter word, word index or domain
 * in either function fails these).
 * ================================================================================== */
enum { DOM_BOND3 = 4 };

static void nbrs3(int64_t L, int64_t i, int64_t nb[6])   /* east, north, up, west, south, down */
{
    int64_t x = i % L, y = (i / L) % L, z = i / (L * L);
    nb[0] = z * L * L + y * L + (x + 1) % L;
    nb[1] = z * L * L + ((y + 1) % L) * L + x;
    nb[2] = ((z + 1) % L) * L * L + y * L + x;
    nb[3] = z * L * L + y * L + (x + L - 1) % L;
    nb[4] = z * L * L + ((y + L - 1) % L) * L + x;
    nb[5] = ((z + L - 1) % L) * L * L + y * L + x;
}

int orc3_init_spins(int32_t L, int32_t q, uint64_t seed, int32_t mode, int8_t *spins)
{
    int64_t N = (int64_t)L * L * L;
    if (L < 3 || q < 2 || q > 8) return -1;
    for (int64_t i = 0; i < N; ++i) {
        uint32_t k = 0;
        if (mode == 1) {
            uint32_t w[4];
            draw(seed, (uint32_t)(i >> 2), 0, DOM_INIT, w);
            k = mulhi_range(w[i & 3], (uint32_t)q);
        }
        spins[i] = store_of(q, k);
    }
    return 0;
}

/* codes[i]: bit 0 east, bit 1 north, bit 2 up.  Returns the number of active bonds. */
int64_t orc3_bonds(int32_t L, uint32_t T, uint64_t seed, uint64_t t, const int8_t *spins, uint8_t *codes)
{
    int64_t N = (int64_t)L * L * L, active = 0;
    for (int64_t i = 0; i < N; ++i) {
        uint32_t w[4];
        int64_t nb[6];
        draw(seed, (uint32_t)i, t, DOM_BOND3, w);
        nbrs3(L, i, nb);
        uint8_t c = 0;
        for (int d = 0; d < 3; ++d)
            if (spins[i] == spins[nb[d]] && w[d] < T) { c |= (uint8_t)(1u << d); ++active; }
        codes[i] = c;
    }
    return active;
}

/* breadth-first search, seeds in increasing order: label = minimum site index */
int64_t orc3_label(int32_t L, const uint8_t *codes, int32_t *labels)
{
    int64_t N = (int64_t)L * L * L, nclusters = 0;
    int32_t *queue = (int32_t *)malloc((size_t)N * sizeof(int32_t));
    if (!queue) return -1;
    for (int64_t i = 0; i < N; ++i) labels[i] = -1;
    for (int64_t seed_site = 0; seed_site < N; ++seed_site) {
        if (labels[seed_site] != -1) continue;
        ++nclusters;
        int64_t head = 0, tail = 0;
        labels[seed_site] = (int32_t)seed_site;
        queue[tail++] = (int32_t)seed_site;
        while (head < tail) {
            int64_t i = queue[head++], nb[6];
            nbrs3(L, i, nb);
            for (int d = 0; d < 3; ++d) {
                /* my own bond in direction d, and the bond of the neighbour behind me in direction d */
                if ((codes[i] >> d) & 1) {
                    int64_t j = nb[d];
                    if (labels[j] == -1) { labels[j] = (int32_t)seed_site; queue[tail++] = (int32_t)j; }
                }
                int64_t j = nb[3 + d];
                if (((codes[j] >> d) & 1) && labels[j] == -1) { labels[j] = (int32_t)seed_site; queue[tail++] = (int32_t)j; }
            }
        }
    }
    free(queue);
    return nclusters;
}

void orc3_flip(int64_t N, int32_t q, uint64_t seed, uint64_t t, const int32_t *labels, int8_t *spins)
{
    for (int64_t i = 0; i < N; ++i) {
        uint32_t w[4];
        draw(seed, (uint32_t)labels[i], t, DOM_FLIP, w);
        spins[i] = store_of(q, mulhi_range(w[0], (uint32_t)q));
    }
}

/* sat counts the 3N bonds; Ising E = -sum s_i s_j = -(2 sat - 3N), Potts E = -sat (Eq. 1) */
void orc3_observables(int32_t L, int32_t q, const int8_t *spins, orc_obs *o)
{
    int64_t N = (int64_t)L * L * L;
    memset(o, 0, sizeof(*o));
    for (int64_t i = 0; i < N; ++i) {
        int64_t nb[6];
        nbrs3(L, i, nb);
        for (int d = 0; d < 3; ++d) o->sat_bonds += (spins[i] == spins[nb[d]]);
        int k = (q == 2) ? (spins[i] == 1 ? 0 : 1) : (int)(uint8_t)spins[i];
        if (k >= 0 && k < 8) o->state_count[k] += 1;
    }
    if (q == 2) {
        o->energy = -(2 * o->sat_bonds - 3 * N);
        o->magnetisation = o->state_count[0] - o->state_count[1];
    } else {
        int64_t mx = 0;
        for (int k = 0; k < q; ++k) if (o->state_count[k] > mx) mx = o->state_count[k];
        o->energy = -o->sat_bonds;
        o->magnetisation = (int64_t)q * mx - N;
    }
}

int64_t orc3_sweep(int32_t L, int32_t q, uint32_t T, uint64_t seed, uint64_t t,
                   int8_t *spins, int32_t *labels, uint8_t *codes, int64_t *active)
{
    int64_t N = (int64_t)L * L * L;
    int own_labels = (labels == NULL), own_codes = (codes == NULL);
    if (own_labels) labels = (int32_t *)malloc((size_t)N * sizeof(int32_t));
    if (own_codes)  codes  = (uint8_t *)malloc((size_t)N);
    if (!labels || !codes) return -1;
    int64_t nb = orc3_bonds(L, T, seed, t, spins, codes);
    int64_t nc = orc3_label(L, codes, labels);
    orc3_flip(N, q, seed, t, labels, spins);
    if (active) *active = nb;
    if (own_labels) free(labels);
    if (own_codes)  free(codes);
    return nc;
}

/* series[4*s + 0..3] = energy, magnetisation, n_clusters, sum of squared cluster sizes */
int orc3_run_chain(int32_t L, int32_t q, uint32_t T, uint64_t seed, uint64_t t0,
                   int64_t n, int8_t *spins, int64_t *series)
{
    int64_t N = (int64_t)L * L * L;
    int32_t *labels = (int32_t *)malloc((size_t)N * sizeof(int32_t));
    uint8_t *codes = (uint8_t *)malloc((size_t)N);
    if (!labels || !codes) return -1;
    for (int64_t s = 0; s < n; ++s) {
        int64_t nb = 0;
        int64_t nc = orc3_sweep(L, q, T, seed, t0 + (uint64_t)s, spins, labels, codes, &nb);
        if (series) {
            orc_obs o; orc_cstats c;
            orc3_observables(L, q, spins, &o);
            orc_cluster_stats(N, labels, &c);
            series[4 * s + 0] = o.energy;
            series[4 * s + 1] = o.magnetisation;
            series[4 * s + 2] = nc;
            series[4 * s + 3] = (int64_t)c.sum_sq_cluster;
        }
    }
    free(labels); free(codes);
    return 0;
}
