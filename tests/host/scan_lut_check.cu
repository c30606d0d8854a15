// Host-side check of k_scan's permutation tables (paper_1105_5804_b200/csrc/scan_kernel.cuh make_scan_lut): for every
// pattern of the lane's east bonds, north contacts and links to the neighbouring lanes, the names produced by the table
// selectors (PRMT emulated on the host) must equal the plain definition -- a site takes the name carried by the leftmost
// contact of its run, else the name of the run's first site; sites of the run that enters from / leaves to the
// neighbouring lane take the run names RP / RS.  Built and run by tests/test_scan_lut_cpu.py (no GPU needed).
#include <cstdint>
#include <cstdio>
#include <cstdlib>

#include "../../paper_1105_5804_b200/csrc/label_kernels.cuh"   // includes scan_kernel.cuh after the helpers it uses

static uint32_t prmt_host(uint32_t a, uint32_t b, uint32_t s)
{
    const uint64_t ab = ((uint64_t)b << 32) | a;
    uint32_t d = 0;
    for (int i = 0; i < 4; ++i) d |= (uint32_t)((ab >> (8 * ((s >> (4 * i)) & 7))) & 0xFF) << (8 * i);
    return d;
}

int main()
{
    static const swb::ScanLut t = swb::make_scan_lut();
    long checked = 0;
    srand(12345);
    for (int e4 = 0; e4 < 16; ++e4)
        for (int np = 0; np < 16; ++np)
            for (int EL = 0; EL < 2; ++EL)
                for (int rep = 0; rep < 8; ++rep) {
                    uint32_t P[4], NEW[4];
                    const uint32_t n0 = (uint32_t)(rand() % 1000) * 4u;
                    for (int j = 0; j < 4; ++j) { P[j] = 0x100u + (uint32_t)(rand() % 3000); NEW[j] = n0 + j; }
                    const uint32_t RP = 0x0F00u + (uint32_t)(rand() % 100), RS = 0x0E00u + (uint32_t)(rand() % 100);
                    const bool E[4] = {(e4 & 1) != 0, (e4 & 2) != 0, (e4 & 4) != 0, (e4 & 8) != 0};
                    // ---- plain definition
                    int s[4] = {0, E[0] ? 0 : 1, 0, 0};
                    s[2] = E[1] ? s[1] : 2;
                    s[3] = E[2] ? s[2] : 3;
                    const bool full = E[0] && E[1] && E[2];
                    const bool useP = EL && !full, useS = E[3] || (full && EL);
                    uint32_t want_pre[4], want[4];
                    bool cs = false, cp = false;
                    for (int j = 0; j < 4; ++j) {
                        int lc = -1;
                        for (int k = 3; k >= 0; --k) if (s[k] == s[j] && ((np >> k) & 1)) lc = k;
                        want_pre[j] = lc >= 0 ? P[lc] : NEW[s[j]];
                        if (j == 3) cs = lc >= 0;
                        if (j == 0) cp = lc >= 0;
                        want[j] = (useS && s[j] == s[3]) ? RS : (useP && s[j] == 0) ? RP : want_pre[j];
                    }
                    // ---- table driven, as in k_scan
                    const uint32_t P01 = P[0] | (P[1] << 16), P23 = P[2] | (P[3] << 16);
                    const uint32_t NEW01 = NEW[0] | (NEW[1] << 16), NEW23 = NEW[2] | (NEW[3] << 16);
                    const int ia = (e4 & 1) | ((e4 & 2) << 1) | ((e4 & 4) << 2) | ((np & 1) << 1) | ((np & 2) << 2) |
                                   ((np & 4) << 3) | ((np & 8) << 3);
                    const uint32_t* A = t.a[ia];
                    const uint32_t X = prmt_host(P01, P23, A[0]);
                    uint32_t l01 = prmt_host(X, NEW01, A[0] >> 16);
                    const uint32_t W = prmt_host(P23, NEW23, A[1]);
                    uint32_t l23 = prmt_host(W, l01, A[1] >> 16);
                    const uint32_t pre[4] = {l01 & 0xFFFF, l01 >> 16, l23 & 0xFFFF, l23 >> 16};
                    const int ib = (e4 & 1) | ((e4 & 2) << 1) | ((e4 & 4) << 2) | ((e4 & 8) << 3) | (EL << 1);
                    const uint32_t RPS = RP | (RS << 16);
                    l01 = prmt_host(l01, RPS, t.b[ib]);
                    l23 = prmt_host(l23, RPS, t.b[ib] >> 16);
                    const uint32_t got[4] = {l01 & 0xFFFF, l01 >> 16, l23 & 0xFFFF, l23 >> 16};
                    const uint32_t m01 = prmt_host(0x0000FFFFu, 0u, A[2]), m23 = prmt_host(0x0000FFFFu, 0u, A[2] >> 16);
                    const uint32_t mask[4] = {m01 & 0xFFFF, m01 >> 16, m23 & 0xFFFF, m23 >> 16};
                    int cnt = 0;
                    for (int k = 0; k < 3; ++k) cnt += E[k];
                    for (int k = 0; k < 4; ++k) cnt += (np >> k) & 1;
                    bool ok = ((A[3] & 1u) != 0) == cs && ((A[3] & 2u) != 0) == cp && (int)(A[3] >> 28) == cnt;
                    for (int j = 0; j < 4; ++j)
                        ok = ok && pre[j] == want_pre[j] && got[j] == want[j] && mask[j] == (((np >> j) & 1) ? 0xFFFFu : 0u);
                    if (!ok) {
                        printf("MISMATCH e4=%d np=%d EL=%d\n", e4, np, EL);
                        return 1;
                    }
                    ++checked;
                }
    printf("scan tables ok: %ld cases\n", checked);
    return 0;
}
