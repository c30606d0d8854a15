// Host-side check of k_scan's row logic (paper_1105_5804_b200/csrc/scan_kernel.cuh: the naming tables and row_local /
// row_final / row_mismatch, PRMT emulated on the host): whole rows of 32 lanes are run through the lane code with random
// bonds and random names carried by the previous row, the flagged pairs are united in a plain union-find, and the resulting
// partition must equal the plain definition -- sites joined by east bonds, a site joined to the name above it by a north
// bond.  Every name a site takes must be a node: a name carried by the previous row, or the index of a site of this row that
// kept its own index.  Built and run by tests/test_scan_lut_cpu.py (no GPU needed).
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <vector>

#include "../../paper_1105_5804_b200/csrc/label_kernels.cuh"   // includes scan_kernel.cuh after the helpers it uses

struct UF {
    std::vector<int> p;
    explicit UF(int n) : p(n) { for (int i = 0; i < n; ++i) p[i] = i; }
    int find(int x) { while (p[x] != x) x = p[x] = p[p[x]]; return x; }
    void unite(int a, int b) { a = find(a); b = find(b); if (a != b) p[a] = b; }
};

static const swb::ScanLut T = swb::make_scan_lut();
static const int ROW = 31;                               // names of this row: ROW * 128 + column (12-bit)
static const int NPREV = 3000;                           // names carried by the previous row are < NPREV

// element ids of the union-finds: [0, NPREV) names of the previous row, NPREV + x = site x of this row
static int elem_of_name(uint32_t name) { return name >= (uint32_t)(ROW * 128) ? NPREV + (int)name - ROW * 128 : (int)name; }

static bool check_row(int nlanes, const uint32_t* G, const uint32_t* Gprev, const uint32_t* P, long& nflags)
{
    const int W = 4 * nlanes;
    uint32_t l01[32], l23[32], toR[32], toL[32], A[32][4], B[32][4];
    for (int k = 0; k < nlanes; ++k) {
        const uint32_t g = G[k] & (k == nlanes - 1 ? 0xBFu : 0xFFu);
        const uint32_t* a = T.a[(g & 0x55u) | (Gprev[k] & 0xAAu)];
        const uint32_t* b = T.b[g & 0x15u];
        for (int i = 0; i < 4; ++i) { A[k][i] = a[i]; B[k][i] = b[i]; }
        const uint32_t P01 = P[4 * k] | (P[4 * k + 1] << 16), P23 = P[4 * k + 2] | (P[4 * k + 3] << 16);
        const uint32_t NEW01 = (uint32_t)(ROW * 128 + 4 * k) * 0x00010001u + 0x00010000u, NEW23 = NEW01 + 0x00020002u;
        swb::row_local(A[k], P01, P23, NEW01, NEW23, l01[k], l23[k], toR[k], toL[k]);
    }
    UF alg(NPREV + 128), def(NPREV + 128);
    uint32_t name[128];
    for (int k = 0; k < nlanes; ++k) {
        const uint32_t fromL = toR[k ? k - 1 : k], fromR = toL[k + 1 < nlanes ? k + 1 : k];   // shuffles clamp at the ends
        const uint32_t P01 = P[4 * k] | (P[4 * k + 1] << 16), P23 = P[4 * k + 2] | (P[4 * k + 3] << 16);
        const uint32_t link = swb::row_final(A[k], B[k], fromL, fromR, k ? (swb::F_LK | swb::F_LC) : 0u, l01[k], l23[k]);
        const uint32_t mm = swb::row_mismatch(A[k], P01, P23, l01[k], l23[k]);
        name[4 * k] = l01[k] & 0xFFFF; name[4 * k + 1] = l01[k] >> 16;
        name[4 * k + 2] = l23[k] & 0xFFFF; name[4 * k + 3] = l23[k] >> 16;
        if (mm & ~0x000F0000u) { printf("mismatch flags outside bits 16..19\n"); return false; }
        for (int j = 0; j < 4; ++j)
            if ((mm >> (16 + j)) & 1) {                  // unite the name of the site with the name above it
                if (!((Gprev[k] >> (2 * j + 1)) & 1)) { printf("flag without a contact\n"); return false; }
                alg.unite(elem_of_name(name[4 * k + j]), elem_of_name(P[4 * k + j]));
                ++nflags;
            }
        if (link) {                                      // unite the names of my first site and of its west neighbour
            if (k == 0) { printf("link flag in lane 0\n"); return false; }
            alg.unite(elem_of_name(name[4 * k]), elem_of_name(name[4 * k - 1]));      // name[4k-1] is final: lane k-1 is done
            ++nflags;
        }
    }
    // every site belongs to the cluster of the name it took; every name is a node
    for (int x = 0; x < W; ++x) {
        const uint32_t n = name[x];
        if (n >= (uint32_t)(ROW * 128)) {
            const int s = (int)n - ROW * 128;
            if (s >= W || s > x || name[s] != n) { printf("site %d took the name %u, which is not a node\n", x, n); return false; }
        } else {
            bool found = false;
            for (int k = 0; k < W; ++k) found = found || (P[k] == n && ((Gprev[k >> 2] >> (2 * (k & 3) + 1)) & 1));
            if (!found) { printf("site %d took %u, not a name of a contact\n", x, n); return false; }
        }
        alg.unite(NPREV + x, elem_of_name(n));
    }
    // the plain definition
    for (int x = 0; x < W; ++x) {
        const uint32_t g = G[x >> 2], gp = Gprev[x >> 2];
        if (((g >> (2 * (x & 3))) & 1) && x + 1 < W) def.unite(NPREV + x, NPREV + x + 1);
        if ((gp >> (2 * (x & 3) + 1)) & 1) def.unite(NPREV + x, (int)P[x]);
    }
    // same partition of the sites and the names they can reach
    std::vector<int> elems;
    for (int x = 0; x < W; ++x) { elems.push_back(NPREV + x); elems.push_back((int)P[x]); }
    for (size_t i = 0; i < elems.size(); ++i)
        for (size_t j = i + 1; j < elems.size(); ++j)
            if ((alg.find(elems[i]) == alg.find(elems[j])) != (def.find(elems[i]) == def.find(elems[j]))) {
                printf("partition differs for elements %d %d\n", elems[i], elems[j]);
                return false;
            }
    return true;
}

int main()
{
    srand(20261104);
    long rows = 0, nflags = 0;
    const double dens[][2] = {{0.5, 0.5}, {0.9, 0.5}, {1.0, 0.3}, {0.3, 0.9}, {0.97, 0.05}, {0.7, 0.0}, {0.0, 1.0}, {1.0, 1.0}, {0.85, 0.2}};
    for (const auto& d : dens)
        for (int pool : {1, 2, 5, 40, 2000})
            for (int nlanes : {32, 1, 2, 5})
                for (int rep = 0; rep < 400; ++rep) {
                    uint32_t G[32], Gp[32], P[128];
                    for (int k = 0; k < nlanes; ++k) {
                        G[k] = Gp[k] = 0;
                        for (int j = 0; j < 4; ++j) {
                            if (rand() < d[0] * RAND_MAX) G[k] |= 1u << (2 * j);
                            if (rand() < 0.5 * RAND_MAX) G[k] |= 2u << (2 * j);            // this row's north bonds: ignored here
                            if (rand() < d[1] * RAND_MAX) Gp[k] |= 2u << (2 * j);
                            if (rand() < 0.5 * RAND_MAX) Gp[k] |= 1u << (2 * j);           // previous row's east bonds: ignored
                            P[4 * k + j] = (uint32_t)(rand() % pool) * (pool > 100 ? 1 : 7);
                        }
                    }
                    if (!check_row(nlanes, G, Gp, P, nflags)) {
                        printf("MISMATCH dens=(%g,%g) pool=%d lanes=%d rep=%d\n", d[0], d[1], pool, nlanes, rep);
                        return 1;
                    }
                    ++rows;
                }
    printf("scan rows ok: %ld rows, %ld flags\n", rows, nflags);
    return 0;
}
