// swb200.cu -- the C-ABI of libswb200.so (include/swb200.h): host-side state, argument checks, kernel launches.
// Every step of the path runs in the kernels of label_kernels.cuh / misc_kernels.cuh; there is no CPU fallback.
#include "../../include/swb200.h"

#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>

#include "common.cuh"
#include "label_kernels.cuh"
#include "misc_kernels.cuh"
#include "wolff_kernel.cuh"
#include "cubic_kernels.cuh"
#include "paper_kernels.cuh"
#include "band_kernels.cuh"

using namespace swb;

struct sw_handle {
    int32_t  dim;              // 2: L x L square lattice; 3: L x L x L simple cubic lattice (sw_create3d)
    int32_t  L, q;
    int64_t  N;
    double   beta;
    uint64_t seed;
    uint64_t t;                // step counter
    uint32_t T;
    Params   p;                // kernel parameters (t_lo/t_hi refreshed per launch)
    // bound device buffers (caller-owned)
    uint32_t* d_spins;
    int32_t*  d_labels;
    uint8_t*  d_bonds;
    uint8_t*  d_work;
    uint8_t*  d_bonds3;            // simple cubic lattice: the bond bytes of the last sweep (N bytes of the workspace)
    // carved from d_work
    Acc*      d_acc;
    unsigned long long* d_wolff;   // WOLFF_RING slots
    int32_t*  d_edgeA;             // (ntx+nty)*L: strip-local roots of last columns / last rows (-1: bond inactive)
    int32_t*  d_edgeB;             // (ntx+nty)*L: strip-local roots of first columns / first rows
    int32_t*  d_size;              // N int32
    SeriesEntry* d_series;         // SERIES_RING entries: (sat, minus) of the configuration each sweep / step started from
    uint64_t  series_lo, series_hi; // counters [lo, hi) whose entries are in the ring
    uint32_t* d_draws;             // draw cache: ntx*nty*TH/4*32 words (scan_kernel.cuh)
    int       wolff_levels;        // 0: label everything; > 0: try frontier growth for that many levels first
    int*      d_wolff_status;      // device flag of the frontier kernel (0 done, 1 gave up)
    bool      draws_valid;         // the cache holds the draws of step draws_t for threshold draws_T
    uint64_t  draws_t;
    uint32_t  draws_T;
    bool      bound;
    int       device;              // CUDA device the bound buffers live on (sw_bind); -1 before
    int       band_rank, nbands;   // multi-GPU row bands (sw_set_band): this handle works on band band_rank of nbands; 0, 1 else
    bool      band_open;           // sw_sweep_band_begin has run, sw_sweep_band_end has not
    const int32_t* last_labels;    // labels buffer written by the LAST sweep / step / sw_label (NULL: none since bind)
    uint64_t  launches;
    char      cuda_err[256];
    // optional per-kernel timing (sw_profile_*)
    bool         prof_on;
    int          prof_n;                                  // sweeps recorded since the last read
    cudaEvent_t* prof_ev;                                 // PROF_MAX * (SW_NPHASE + 1) events, created on enable
};

namespace {

constexpr size_t ALIGN = 256;
inline size_t align_up(size_t x) { return (x + ALIGN - 1) / ALIGN * ALIGN; }

struct WorkLayout { size_t acc, wolff, wstatus, series, edgeA, edgeB, draws, size, bonds3, total; };

WorkLayout work_layout(int32_t L, int32_t dim)
{
    const size_t N = dim == 3 ? (size_t)L * L * L : (size_t)L * L;
    // (the cubic path has no strips: no edge arrays, no draw cache; it keeps one bond byte per site)
    const size_t ntx = dim == 3 ? 0 : (L + TW - 1) / TW, nty = dim == 3 ? 0 : (L + TH - 1) / TH;
    WorkLayout w;
    w.acc = 0;
    w.wolff = align_up(sizeof(Acc));
    w.wstatus = w.wolff + align_up(sizeof(unsigned long long) * WOLFF_RING);
    w.series = w.wstatus + align_up(sizeof(int));
    w.edgeA = w.series + align_up(sizeof(SeriesEntry) * SERIES_RING);
    w.edgeB = w.edgeA + align_up((ntx + nty) * (size_t)L * sizeof(int32_t));
    w.draws = w.edgeB + align_up((ntx + nty) * (size_t)L * sizeof(int32_t));
    // (the draw cache exists only in a build with SWB_GEN_ROWS > 0 -- measured and dropped; 64 MiB at L = 16384)
    w.size = w.draws + align_up(GEN_ROWS > 0 ? ntx * nty * (size_t)(TH / 4) * 32 * sizeof(uint32_t) : 0);
    w.bonds3 = w.size + align_up(N * sizeof(int32_t));
    w.total = w.bonds3 + align_up(dim == 3 ? N : 0);
    return w;
}

// labels are < N <= 2^30; k_final packs the new state (q <= 8: 3 bits) above the label, which needs N <= 2^28 unless q = 2
bool valid_shape(int32_t L, int32_t q)
{
    return L >= 4 && L <= 32768 && (L % 4) == 0 && q >= 2 && q <= 8 && (q == 2 || L <= 16384);
}
// simple cubic lattice: N = L^3 <= 2^30 (site indices and labels are int32)
bool valid_shape3(int32_t L, int32_t q)
{
    return L >= 4 && L <= 1024 && (L % 4) == 0 && q >= 2 && q <= 8;
}

// Every entry point that launches or copies makes the device of the bound buffers current for the call (a caller with
// several GPUs need not have it current) and restores the previous one.
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    explicit DeviceGuard(const sw_handle* h)
    {
        if (h && h->device >= 0 && cudaGetDevice(&prev) == cudaSuccess && prev != h->device)
            switched = cudaSetDevice(h->device) == cudaSuccess;
    }
    ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};

int cuda_fail(sw_handle* h, cudaError_t e, const char* where)
{
    if (h) snprintf(h->cuda_err, sizeof(h->cuda_err), "%s: %s", where, cudaGetErrorString(e));
    return SW_ECUDA;
}

#define SW_CUDA(h, call)                                                     \
    do {                                                                     \
        cudaError_t e__ = (call);                                            \
        if (e__ != cudaSuccess) return cuda_fail((h), e__, #call);           \
    } while (0)

#define SW_LAUNCHED(h, name)                                                 \
    do {                                                                     \
        cudaError_t e__ = cudaGetLastError();                                \
        if (e__ != cudaSuccess) return cuda_fail((h), e__, name);            \
        ++(h)->launches;                                                     \
    } while (0)

uint32_t threshold_of(int32_t q, double beta)
{
    // S:8c.4 / reading 6: floor((1 - exp(-K beta)) 2^32) in IEEE double, K = 2 for q = 2 (Ising +-1), else 1
    const double K = (q == 2) ? 2.0 : 1.0;
    double v = std::floor((1.0 - std::exp(-K * beta)) * 4294967296.0);
    if (v < 0.0) v = 0.0;
    if (v > 4294967295.0) v = 4294967295.0;
    return (uint32_t)v;
}

Params params_at(const sw_handle* h, uint64_t t)
{
    Params p = h->p;
    p.T = h->T;
    p.negT = 0u - h->T;
    p.dmask = h->T ? 0xFFu : 0u;
    p.t_lo = (uint32_t)(t & 0xFFFFFFFFu);
    p.t_hi = (uint32_t)(t >> 32);
    p.u_lo = (uint32_t)((t + 1) & 0xFFFFFFFFu);
    p.u_hi = (uint32_t)((t + 1) >> 32);
    return p;
}

constexpr int PROF_MAX = 512;
inline int prof_mark(sw_handle* h, int phase, cudaStream_t s)
{
    if (h->prof_on && h->prof_n < PROF_MAX)
        SW_CUDA(h, cudaEventRecord(h->prof_ev[h->prof_n * (SW_NPHASE + 1) + phase], s));
    return SW_OK;
}
#define SW_PROF(h, phase, s)                                                 \
    do {                                                                     \
        int rc__ = prof_mark((h), (phase), (s));                             \
        if (rc__) return rc__;                                               \
    } while (0)

inline int grid_for(int64_t n, int block) { return (int)((n + block - 1) / block); }
inline int grid_capped(int64_t n, int block, int cap) { int g = grid_for(n, block); return g < cap ? (g < 1 ? 1 : g) : cap; }

#if SWB_PDL == 2
// the per-sweep counters are zeroed by a kernel, so that the chain k_final -> k_zero -> k_scan is kernel to kernel
__global__ void k_zero(Acc* acc)
{
    cudaGridDependencySynchronize();
    reinterpret_cast<uint4*>(acc->part)[threadIdx.x] = make_uint4(0u, 0u, 0u, 0u);
}
inline cudaLaunchAttribute pdl_attr()
{
    cudaLaunchAttribute a;
    a.id = cudaLaunchAttributeProgrammaticStreamSerialization; a.val.programmaticStreamSerializationAllowed = 1;
    return a;
}
#endif

// A kernel that asks for more dynamic shared memory than the 48 KB default needs cudaFuncAttributeMaxDynamicSharedMemorySize
// raised -- a property of the kernel ON ONE DEVICE.  The (device, kernel) pairs already done are remembered; the default
// build (SCAN_WARPS = 4: ScanSmem is 37.9 KB) never gets past the first line.  The device of the handle is current here.
int raise_smem_limit(sw_handle* h, const void* kern, int bytes)
{
    if (bytes <= 48 * 1024) return SW_OK;
    struct Done { int dev; const void* kern; };
    static std::mutex mtx;
    static Done done[256];
    static int ndone = 0;
    int dev = 0;
    SW_CUDA(h, cudaGetDevice(&dev));
    std::lock_guard<std::mutex> lock(mtx);
    for (int i = 0; i < ndone; ++i) if (done[i].dev == dev && done[i].kern == kern) return SW_OK;
    SW_CUDA(h, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
    if (ndone < 256) done[ndone++] = Done{dev, kern};    // (a full table only means the attribute is set again next time)
    return SW_OK;
}

// labelling of the bond graph of step t (or of packed bonds): k_scan -> k_seam; k_final resolves the rest
// SRC_PHILOX falls through to SRC_DRAWS when the draw cache holds the draws of step t for the current threshold
template <int SRC>
int launch_label_front(sw_handle* h, const Params& p, const uint8_t* bonds, int32_t* labels, cudaStream_t s,
                       bool record_series = false)
{
    SW_PROF(h, 0, s);
    const dim3 grid((p.ntx + SCAN_WARPS - 1) / SCAN_WARPS, p.nband);      // (nband = nty unless the handle works on a row band)
    auto seam = h->nbands > 1 ? k_seam<true> : k_seam<false>;
    const bool ising = SRC == SRC_BONDS || p.q == 2, fullw = (p.L % TW) == 0;
    const uint64_t t = ((uint64_t)p.t_hi << 32) | p.t_lo;
    const bool cached = SRC == SRC_PHILOX && h->draws_valid && h->draws_t == t && h->draws_T == h->T;
    auto kern = SRC == SRC_BONDS ? (fullw ? k_scan<SRC_BONDS, true, true> : k_scan<SRC_BONDS, true, false>)
              : cached ? (ising ? (fullw ? k_scan<SRC_DRAWS, true, true> : k_scan<SRC_DRAWS, true, false>)
                                : (fullw ? k_scan<SRC_DRAWS, false, true> : k_scan<SRC_DRAWS, false, false>))
                       : (ising ? (fullw ? k_scan<SRC_PHILOX, true, true> : k_scan<SRC_PHILOX, true, false>)
                                : (fullw ? k_scan<SRC_PHILOX, false, true> : k_scan<SRC_PHILOX, false, false>));
    if (h->nbands > 1)                                   // a row band: L is a multiple of TH, sweeps only (no draw cache)
        kern = ising ? (fullw ? k_scan<SRC_PHILOX, true, true, true> : k_scan<SRC_PHILOX, true, false, true>)
                     : (fullw ? k_scan<SRC_PHILOX, false, true, true> : k_scan<SRC_PHILOX, false, false, true>);
    {
        const int rc = raise_smem_limit(h, (const void*)kern, (int)sizeof(ScanSmem));
        if (rc) return rc;
    }
#if SWB_PDL == 2
    {
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = grid; cfg.blockDim = dim3(SCAN_THREADS); cfg.dynamicSmemBytes = sizeof(ScanSmem); cfg.stream = s;
        cudaLaunchAttribute at[1] = {pdl_attr()};
        cfg.attrs = at; cfg.numAttrs = 1;
        SW_CUDA(h, cudaLaunchKernelEx(&cfg, kern, p, (const uint32_t*)h->d_spins, bonds, (const uint32_t*)h->d_draws, (int*)labels,
                                      (int*)h->d_edgeA, (int*)h->d_edgeB, h->d_acc));
    }
#else
    kern<<<grid, SCAN_THREADS, sizeof(ScanSmem), s>>>(p, h->d_spins, bonds, h->d_draws, labels, h->d_edgeA, h->d_edgeB,
                                                      h->d_acc);
#endif
    SW_LAUNCHED(h, "k_scan");
    SW_PROF(h, 1, s);
    const int nseam = h->nbands > 1 ? seam_band_sites(p) : (p.ntx + p.nty) * p.L;
#if SWB_PDL
    {
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(grid_for(seam_part(nseam), 256)); cfg.blockDim = dim3(256); cfg.stream = s;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization; at[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        SW_CUDA(h, cudaLaunchKernelEx(&cfg, seam, p, (const int*)h->d_edgeA, (const int*)h->d_edgeB, (int*)labels,
                                      (const Acc*)h->d_acc, record_series ? h->d_series : (SeriesEntry*)nullptr));
    }
#else
    seam<<<grid_for(seam_part(nseam), 256), 256, 0, s>>>(p, h->d_edgeA, h->d_edgeB, labels, h->d_acc,
                                                          record_series ? h->d_series : nullptr);
#endif
    SW_LAUNCHED(h, "k_seam");
    if (record_series) {                                 // the ring now holds the entry of counter t
        if (t != h->series_hi) h->series_lo = t;
        h->series_hi = t + 1;
        if (h->series_hi - h->series_lo > (uint64_t)SERIES_RING) h->series_lo = h->series_hi - SERIES_RING;
    }
    SW_PROF(h, 2, s);
    return SW_OK;
}

// flatten + flip of a sweep (k_final<MODE_SW>) over the strip rows the handle works on
int launch_final_sw(sw_handle* h, const Params& p, cudaStream_t s)
{
    const bool full = (p.L % TW) == 0 && (p.L % TH) == 0, q2 = p.q == 2;
    auto fin = full ? (q2 ? k_final<MODE_SW, GEN_ROWS, true, true> : k_final<MODE_SW, GEN_ROWS, true, false>)
                    : (q2 ? k_final<MODE_SW, GEN_ROWS, false, true> : k_final<MODE_SW, GEN_ROWS, false, false>);
    if (h->nbands > 1)
        fin = full ? (q2 ? k_final<MODE_SW, GEN_ROWS, true, true, true> : k_final<MODE_SW, GEN_ROWS, true, false, true>)
                   : (q2 ? k_final<MODE_SW, GEN_ROWS, false, true, true> : k_final<MODE_SW, GEN_ROWS, false, false, true>);
#if SWB_PDL
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(p.ntx, p.nband); cfg.blockDim = dim3(FIN_THREADS); cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization; at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    SW_CUDA(h, cudaLaunchKernelEx(&cfg, fin, p, (int*)h->d_labels, h->d_spins, h->d_acc, (unsigned long long*)nullptr, h->d_draws));
#else
    fin<<<dim3(p.ntx, p.nband), FIN_THREADS, 0, s>>>(p, h->d_labels, h->d_spins, h->d_acc, nullptr, h->d_draws);
#endif
    SW_LAUNCHED(h, "k_final<SW>");
    return SW_OK;
}

int zero_sweep_counters(sw_handle* h, cudaStream_t s)
{
#if SWB_PDL == 2
    static_assert(sizeof(AccPart) * ACC_PARTS == 256 * sizeof(uint4), "k_zero: one uint4 per thread");
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(1); cfg.blockDim = dim3(256); cfg.stream = s;
    cudaLaunchAttribute at[1] = {pdl_attr()};
    cfg.attrs = at; cfg.numAttrs = 1;
    SW_CUDA(h, cudaLaunchKernelEx(&cfg, k_zero, h->d_acc));
    ++h->launches;
#else
    // the per-sweep counters (n_active, n_clusters) are the parts at the start of Acc
    SW_CUDA(h, cudaMemsetAsync(h->d_acc, 0, sizeof(AccPart) * ACC_PARTS, s));
#endif
    return SW_OK;
}

}  // namespace

extern "C" {

const char* sw_strerror(int code)
{
    switch (code) {
        case SW_OK: return "ok";
        case SW_EINVAL: return "invalid argument";
        case SW_ESTATE: return "handle not bound, or a needed buffer was bound as NULL";
        case SW_ECUDA: return "CUDA error (see sw_last_cuda_error)";
        case SW_ENOMEM: return "out of host memory";
        case SW_ELIMIT: return "lattice larger than the built-in scratch array (SW_STATIC_MAX_SITES sites): use sw_cluster_stats with a workspace";
        default: return "unknown error code";
    }
}

const char* sw_last_cuda_error(const sw_handle* h) { return h ? h->cuda_err : ""; }

static int create_any(sw_handle** out, int32_t dim, int32_t L, int32_t q, double beta, uint64_t seed)
{
    if (!out) return SW_EINVAL;
    *out = nullptr;
    if (!(dim == 3 ? valid_shape3(L, q) : valid_shape(L, q)) || !std::isfinite(beta) || beta < 0.0) return SW_EINVAL;
    sw_handle* h = new (std::nothrow) sw_handle;
    if (!h) return SW_ENOMEM;
    memset(h, 0, sizeof(*h));
    h->dim = dim;
    h->device = -1;
    h->L = L; h->q = q; h->N = dim == 3 ? (int64_t)L * L * L : (int64_t)L * L; h->beta = beta; h->seed = seed; h->t = 0;
    h->T = threshold_of(q, beta);
    Params& p = h->p;
    p.L = L; p.N = (int32_t)h->N; p.q = q;
    p.logL = -1;
    p.sbit = h->N <= (1 << 28) ? 28 : 30;
    for (int k = 2; k <= 15; ++k) if ((1 << k) == L) p.logL = k;
    p.ntx = (L + TW - 1) / TW; p.nty = (L + TH - 1) / TH;
    p.ty0 = 0; p.nband = p.nty;
    h->band_rank = 0; h->nbands = 1;
    p.H = L;
    if (dim == 3) {
        p.H = L * L; p.nty = (p.H + TH - 1) / TH;        // (label array as L*L rows of L sites: cluster statistics)
        p.n3x = (L + C3X - 1) / C3X; p.n3y = (L + C3Y - 1) / C3Y; p.n3z = (L + C3Z - 1) / C3Z;
    }
    const uint32_t s_lo = (uint32_t)(seed & 0xFFFFFFFFu), s_hi = (uint32_t)(seed >> 32);
    for (int r = 0; r < 10; ++r) {
        p.k0[r] = s_lo + (uint32_t)r * 0x9E3779B9u;
        p.k1[r] = s_hi + (uint32_t)r * 0xBB67AE85u;
    }
    *out = h;
    return SW_OK;
}

int sw_create(sw_handle** out, int32_t L, int32_t q, double beta, uint64_t seed) { return create_any(out, 2, L, q, beta, seed); }
int sw_create3d(sw_handle** out, int32_t L, int32_t q, double beta, uint64_t seed) { return create_any(out, 3, L, q, beta, seed); }

int sw_profile_enable(sw_handle* h, int on)
{
    if (!h) return SW_EINVAL;
    DeviceGuard guard(h);
    if (on && !h->prof_ev) {
        h->prof_ev = new (std::nothrow) cudaEvent_t[PROF_MAX * (SW_NPHASE + 1)];
        if (!h->prof_ev) return SW_ENOMEM;
        for (int i = 0; i < PROF_MAX * (SW_NPHASE + 1); ++i) SW_CUDA(h, cudaEventCreate(&h->prof_ev[i]));
    }
    h->prof_on = on != 0;
    h->prof_n = 0;
    return SW_OK;
}

int sw_profile_read(sw_handle* h, double ms[SW_NPHASE], uint64_t* n_sweeps)
{
    if (!h || !ms || !n_sweeps) return SW_EINVAL;
    if (!h->prof_ev) return SW_ESTATE;
    DeviceGuard guard(h);
    for (int k = 0; k < h->prof_n; ++k) {
        cudaEvent_t* e = h->prof_ev + k * (SW_NPHASE + 1);
        SW_CUDA(h, cudaEventSynchronize(e[SW_NPHASE]));
        for (int ph = 0; ph < SW_NPHASE; ++ph) {
            float t = 0.f;
            SW_CUDA(h, cudaEventElapsedTime(&t, e[ph], e[ph + 1]));
            ms[ph] += (double)t;
        }
    }
    *n_sweeps += (uint64_t)h->prof_n;
    h->prof_n = 0;
    return SW_OK;
}

int sw_destroy(sw_handle* h)
{
    if (!h) return SW_EINVAL;
    if (h->prof_ev) {
        for (int i = 0; i < PROF_MAX * (SW_NPHASE + 1); ++i) cudaEventDestroy(h->prof_ev[i]);
        delete[] h->prof_ev;
    }
    delete h;
    return SW_OK;
}

size_t sw_workspace_bytes(int32_t L, int32_t q)
{
    if (!valid_shape(L, q)) return 0;
    return work_layout(L, 2).total;
}

size_t sw_workspace_bytes3d(int32_t L, int32_t q)
{
    if (!valid_shape3(L, q)) return 0;
    return work_layout(L, 3).total;
}

int sw_bind(sw_handle* h, void* d_spins, int32_t* d_labels, uint8_t* d_bonds, void* d_work, size_t work_bytes,
            void* stream)
{
    if (!h || !d_spins || !d_labels || !d_work) return SW_EINVAL;
    if (((uintptr_t)d_spins | (uintptr_t)d_labels | (uintptr_t)d_bonds | (uintptr_t)d_work) & 15u) return SW_EINVAL;
    const WorkLayout w = work_layout(h->L, h->dim);
    if (work_bytes < w.total) return SW_EINVAL;
    {   // the device the buffers live on (a pointer that is not device memory is refused)
        cudaPointerAttributes at;
        if (cudaPointerGetAttributes(&at, d_spins) != cudaSuccess || (at.type != cudaMemoryTypeDevice && at.type != cudaMemoryTypeManaged)) {
            cudaGetLastError();
            return SW_EINVAL;
        }
        h->device = at.device;
    }
    DeviceGuard guard(h);
    h->d_spins = (uint32_t*)d_spins;
    h->d_labels = d_labels;
    h->d_bonds = d_bonds;
    h->d_work = (uint8_t*)d_work;
    h->d_acc = (Acc*)(h->d_work + w.acc);
    h->d_wolff = (unsigned long long*)(h->d_work + w.wolff);
    h->d_edgeA = (int32_t*)(h->d_work + w.edgeA);
    h->d_edgeB = (int32_t*)(h->d_work + w.edgeB);
    h->d_size = (int32_t*)(h->d_work + w.size);
    h->d_bonds3 = h->d_work + w.bonds3;
    h->d_draws = (uint32_t*)(h->d_work + w.draws);
    h->d_series = (SeriesEntry*)(h->d_work + w.series);
    h->d_wolff_status = (int*)(h->d_work + w.wstatus);
    h->series_lo = h->series_hi = 0;
    h->draws_valid = false;
    h->bound = false;
    h->last_labels = nullptr;
    SW_CUDA(h, cudaMemsetAsync(h->d_work, 0, w.edgeA, (cudaStream_t)stream));
    h->bound = true;
    return SW_OK;
}

int sw_set_threshold(sw_handle* h, uint32_t T) { if (!h) return SW_EINVAL; h->T = T; return SW_OK; }
int sw_get_threshold(const sw_handle* h, uint32_t* T) { if (!h || !T) return SW_EINVAL; *T = h->T; return SW_OK; }
int sw_set_counter(sw_handle* h, uint64_t t) { if (!h) return SW_EINVAL; h->t = t; return SW_OK; }
int sw_get_counter(const sw_handle* h, uint64_t* t) { if (!h || !t) return SW_EINVAL; *t = h->t; return SW_OK; }
int sw_launch_count(const sw_handle* h, uint64_t* n) { if (!h || !n) return SW_EINVAL; *n = h->launches; return SW_OK; }

int sw_init_spins(sw_handle* h, int mode, void* stream)
{
    if (!h || (mode != 0 && mode != 1)) return SW_EINVAL;
    if (!h->bound) return SW_ESTATE;
    DeviceGuard guard(h);
    const Params p = params_at(h, 0);
    k_init<<<grid_capped(h->N / 4, 256, 148 * 16), 256, 0, (cudaStream_t)stream>>>(p, h->d_spins, mode);
    SW_LAUNCHED(h, "k_init");
    return SW_OK;
}

// one sweep of the simple cubic lattice (cubic_kernels.cuh): k3_local -> k3_faces -> k3_final
static int sweep3(sw_handle* h, cudaStream_t s)
{
    const Params p = params_at(h, h->t);
    int rc = zero_sweep_counters(h, s);
    if (rc) return rc;
    const int ntiles = p.n3x * p.n3y * p.n3z;
    const int gw = grid_capped(h->N / 4, 256, 148 * 16);
    SW_PROF(h, 0, s);
    if (h->q == 2) k3_local<true><<<ntiles, C3THREADS, 0, s>>>(p, h->d_spins, h->d_labels, h->d_bonds3, h->d_acc);
    else           k3_local<false><<<ntiles, C3THREADS, 0, s>>>(p, h->d_spins, h->d_labels, h->d_bonds3, h->d_acc);
    SW_LAUNCHED(h, "k3_local");
    SW_PROF(h, 1, s);
    k3_faces<<<(unsigned)((faces3_ids(h->L) + 255) / 256), 256, 0, s>>>(p, h->d_bonds3, h->d_labels, h->d_acc, h->d_series);
    SW_LAUNCHED(h, "k3_faces");
    if (h->t != h->series_hi) h->series_lo = h->t;
    h->series_hi = h->t + 1;
    if (h->series_hi - h->series_lo > (uint64_t)SERIES_RING) h->series_lo = h->series_hi - SERIES_RING;
    SW_PROF(h, 2, s);
    if (h->q == 2) k3_final<true><<<gw, 256, 0, s>>>(p, h->d_labels, h->d_spins, h->d_acc);
    else           k3_final<false><<<gw, 256, 0, s>>>(p, h->d_labels, h->d_spins, h->d_acc);
    SW_LAUNCHED(h, "k3_final");
    SW_PROF(h, 3, s);
    if (h->prof_on && h->prof_n < PROF_MAX) ++h->prof_n;
    ++h->t;
    h->last_labels = h->d_labels;
    return SW_OK;
}

// ---- multi-GPU row bands (band_kernels.cuh) -----------------------------------------------------------------------------
int sw_set_band(sw_handle* h, int rank, int nranks)
{
    if (!h || h->dim != 2 || nranks < 1 || rank < 0 || rank >= nranks) return SW_EINVAL;
    if (h->p.nty % nranks != 0 || (h->L % TH) != 0) return SW_EINVAL;      // uniform bands of whole strip rows
    h->band_rank = rank; h->nbands = nranks; h->band_open = false;
    h->p.nband = h->p.nty / nranks;
    h->p.ty0 = rank * h->p.nband;
    return SW_OK;
}

int sw_band_layout(const sw_handle* h, int band, int32_t* y_first, int32_t* n_rows, int32_t* y_halo,
                   size_t* work_off_rootN, size_t* work_off_rootS)
{
    if (!h || band < 0 || band >= h->nbands) return SW_EINVAL;
    const int nb = h->p.nty / h->nbands, L = h->L;
    const WorkLayout w = work_layout(h->L, h->dim);
    const size_t nE = (size_t)h->p.ntx * L;
    if (y_first) *y_first = band * nb * TH;
    if (n_rows) *n_rows = nb * TH;
    if (y_halo) *y_halo = ((band + 1) * nb * TH) % L;
    if (work_off_rootN) *work_off_rootN = w.edgeA + (nE + (size_t)((band + 1) * nb - 1) * L) * sizeof(int32_t);
    if (work_off_rootS) *work_off_rootS = w.edgeB + (nE + (size_t)(band * nb) * L) * sizeof(int32_t);
    return SW_OK;
}

int sw_sweep_band_begin(sw_handle* h, void* stream)
{
    if (!h) return SW_EINVAL;
    if (!h->bound || h->nbands < 2 || h->band_open) return SW_ESTATE;
    DeviceGuard guard(h);
    cudaStream_t s = (cudaStream_t)stream;
    const Params p = params_at(h, h->t);
    int rc = zero_sweep_counters(h, s);
    if (rc) return rc;
    rc = launch_label_front<SRC_PHILOX>(h, p, nullptr, h->d_labels, s, false);
    if (rc) return rc;
    k_band_resolve<<<grid_for(p.L, 256), 256, 0, s>>>(p, h->d_edgeA, h->d_edgeB, h->d_labels);
    SW_LAUNCHED(h, "k_band_resolve");
    h->band_open = true;
    return SW_OK;
}

int sw_sweep_band_end(sw_handle* h, void* stream)
{
    if (!h) return SW_EINVAL;
    if (!h->bound || h->nbands < 2 || !h->band_open) return SW_ESTATE;
    DeviceGuard guard(h);
    cudaStream_t s = (cudaStream_t)stream;
    const Params p = params_at(h, h->t);
    const int g = grid_for((int64_t)h->nbands * p.L, 256);
    k_band_init<<<g, 256, 0, s>>>(p, h->d_edgeA, h->d_edgeB, h->d_labels, h->nbands);
    SW_LAUNCHED(h, "k_band_init");
    k_band_cross<<<g, 256, 0, s>>>(p, h->d_edgeA, h->d_edgeB, h->d_labels, h->nbands);
    SW_LAUNCHED(h, "k_band_cross");
    const int rc = launch_final_sw(h, p, s);
    if (rc) return rc;
    h->band_open = false;
    h->series_lo = h->series_hi = h->t + 1;               // (the series counters cover a band only: not kept)
    ++h->t;
    h->last_labels = h->d_labels;
    return SW_OK;
}

int sw_band_counters(sw_handle* h, int64_t h_out[4], void* stream)
{
    if (!h || !h_out) return SW_EINVAL;
    if (!h->bound) return SW_ESTATE;
    DeviceGuard guard(h);
    cudaStream_t s = (cudaStream_t)stream;
    Acc a;
    SW_CUDA(h, cudaMemcpyAsync(&a, h->d_acc, sizeof(AccPart) * ACC_PARTS, cudaMemcpyDeviceToHost, s));
    SW_CUDA(h, cudaStreamSynchronize(s));
    h_out[0] = h_out[1] = h_out[2] = h_out[3] = 0;
    for (int k = 0; k < ACC_PARTS; ++k) {
        h_out[0] += (int64_t)a.part[k].n_active; h_out[1] += (int64_t)a.part[k].n_clusters;
        h_out[2] += (int64_t)a.part[k].sat;      h_out[3] += (int64_t)a.part[k].minus;
    }
    return SW_OK;
}

int sw_sweep(sw_handle* h, int64_t n, void* stream)
{
    if (!h || n < 0) return SW_EINVAL;
    if (!h->bound || h->nbands > 1) return SW_ESTATE;    // a banded handle sweeps through sw_sweep_band_begin / _end
    DeviceGuard guard(h);
    cudaStream_t s = (cudaStream_t)stream;
    if (h->dim == 3) {
        for (int64_t k = 0; k < n; ++k) {
            const int rc = sweep3(h, s);
            if (rc) return rc;
        }
        return SW_OK;
    }
    for (int64_t k = 0; k < n; ++k) {
        const Params p = params_at(h, h->t);
        int rc = zero_sweep_counters(h, s);
        if (rc) return rc;
        rc = launch_label_front<SRC_PHILOX>(h, p, nullptr, h->d_labels, s, true);
        if (rc) return rc;
        rc = launch_final_sw(h, p, s);
        if (rc) return rc;
        h->draws_valid = GEN_ROWS > 0; h->draws_t = h->t + 1; h->draws_T = h->T;
        SW_PROF(h, 3, s);
        if (h->prof_on && h->prof_n < PROF_MAX) ++h->prof_n;
        ++h->t;
        h->last_labels = h->d_labels;
    }
    return SW_OK;
}

int sw_activate(sw_handle* h, void* stream)
{
    if (!h) return SW_EINVAL;
    if (!h->bound || !h->d_bonds || h->nbands > 1) return SW_ESTATE;
    DeviceGuard guard(h);
    const Params p = params_at(h, h->t);
    if (h->dim == 3) {                                   // one byte per site: bit 0 east, 1 north, 2 up
        const int gw = grid_capped(h->N / 4, 256, 148 * 16);
        if (h->q == 2) k3_activate<true><<<gw, 256, 0, (cudaStream_t)stream>>>(p, h->d_spins, h->d_bonds);
        else           k3_activate<false><<<gw, 256, 0, (cudaStream_t)stream>>>(p, h->d_spins, h->d_bonds);
        SW_LAUNCHED(h, "k3_activate");
        return SW_OK;
    }
    if (h->q == 2)
        k_activate<true><<<grid_capped(h->N / 16, 256, 148 * 16), 256, 0, (cudaStream_t)stream>>>(p, h->d_spins, h->d_bonds);
    else
        k_activate<false><<<grid_capped(h->N / 16, 256, 148 * 16), 256, 0, (cudaStream_t)stream>>>(p, h->d_spins, h->d_bonds);
    SW_LAUNCHED(h, "k_activate");
    return SW_OK;
}

// sw_label on a cubic handle: one bond byte per site (bits 0-2) -> canonical labels
static int label3(sw_handle* h, const uint8_t* bonds, int32_t* labels, cudaStream_t s)
{
    const Params p = params_at(h, h->t);
    int rc = zero_sweep_counters(h, s);
    if (rc) return rc;
    k3_local<true, true><<<p.n3x * p.n3y * p.n3z, C3THREADS, 0, s>>>(p, nullptr, labels, h->d_bonds3, h->d_acc, bonds);
    SW_LAUNCHED(h, "k3_local<bonds>");
    k3_faces<<<(unsigned)((faces3_ids(h->L) + 255) / 256), 256, 0, s>>>(p, h->d_bonds3, labels, h->d_acc, nullptr);
    SW_LAUNCHED(h, "k3_faces");
    k3_final<true, false><<<grid_capped(h->N / 4, 256, 148 * 16), 256, 0, s>>>(p, labels, nullptr, h->d_acc);
    SW_LAUNCHED(h, "k3_final<labels>");
    h->last_labels = labels;
    return SW_OK;
}

int sw_label(sw_handle* h, const uint8_t* d_bonds_in, int32_t* d_labels_out, void* stream)
{
    if (!h) return SW_EINVAL;
    if (!h->bound) return SW_ESTATE;
    DeviceGuard guard(h);
    if (h->nbands > 1) return SW_ESTATE;
    if (h->dim == 3) {
        const uint8_t* b3 = d_bonds_in ? d_bonds_in : h->d_bonds;
        int32_t* l3 = d_labels_out ? d_labels_out : h->d_labels;
        if (!b3) return SW_ESTATE;
        if (((uintptr_t)b3 | (uintptr_t)l3) & 15u) return SW_EINVAL;
        return label3(h, b3, l3, (cudaStream_t)stream);
    }
    const uint8_t* bonds = d_bonds_in ? d_bonds_in : h->d_bonds;
    int32_t* labels = d_labels_out ? d_labels_out : h->d_labels;
    if (!bonds) return SW_ESTATE;
    if (((uintptr_t)bonds | (uintptr_t)labels) & 15u) return SW_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    const Params p = params_at(h, h->t);
    int rc = zero_sweep_counters(h, s);
    if (rc) return rc;
    rc = launch_label_front<SRC_BONDS>(h, p, bonds, labels, s);
    if (rc) return rc;
    if ((p.L % TW) == 0 && (p.L % TH) == 0)
        k_final<MODE_LABEL, 0, true, true><<<dim3(p.ntx, p.nty), FIN_THREADS, 0, s>>>(p, labels, nullptr, h->d_acc, nullptr, nullptr);
    else
        k_final<MODE_LABEL, 0, false, true><<<dim3(p.ntx, p.nty), FIN_THREADS, 0, s>>>(p, labels, nullptr, h->d_acc, nullptr, nullptr);
    SW_LAUNCHED(h, "k_final<LABEL>");
    SW_PROF(h, 3, s);
    if (h->prof_on && h->prof_n < PROF_MAX) ++h->prof_n;
    h->last_labels = labels;
    return SW_OK;
}

static int cluster_stats_device(sw_handle* h, const int32_t* labels, cudaStream_t s)
{
    const Params p = params_at(h, h->t);
    // (zeroing only the roots' entries from k_cluster_stats instead of this memset was measured: 35 M scattered 4-byte stores
    // take 13 ms -- 2.06 -> 15.6 ms per call; counting the four smallest histogram bins in registers changes nothing)
    SW_CUDA(h, cudaMemsetAsync(h->d_size, 0, (size_t)h->N * sizeof(int32_t), s));
    SW_CUDA(h, cudaMemsetAsync(&h->d_acc->cs_nclusters, 0, sizeof(unsigned long long) * (3 + 32), s));
    k_cluster_sizes<<<dim3(p.ntx, p.nty), 256, 0, s>>>(p, labels, h->d_size);
    SW_LAUNCHED(h, "k_cluster_sizes");
    k_cluster_stats<<<grid_capped(h->N, 256, 148 * 8), 256, 0, s>>>(p, labels, h->d_size, h->d_acc);
    SW_LAUNCHED(h, "k_cluster_stats");
    return SW_OK;
}

int sw_cluster_stats(sw_handle* h, const int32_t* d_labels_in, sw_cstats* h_out, void* stream)
{
    if (!h || !h_out) return SW_EINVAL;
    if (!h->bound || (h->nbands > 1 && !d_labels_in)) return SW_ESTATE;
    DeviceGuard guard(h);
    const int32_t* labels = d_labels_in ? d_labels_in : h->d_labels;
    if ((uintptr_t)labels & 15u) return SW_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    int rc = cluster_stats_device(h, labels, s);
    if (rc) return rc;
    Acc a;
    SW_CUDA(h, cudaMemcpyAsync(&a, h->d_acc, sizeof(Acc), cudaMemcpyDeviceToHost, s));
    SW_CUDA(h, cudaStreamSynchronize(s));
    h_out->n_clusters = (int64_t)a.cs_nclusters;
    h_out->max_cluster = (int64_t)a.cs_max;
    h_out->sum_sq_cluster = a.cs_sumsq;
    for (int b = 0; b < 32; ++b) h_out->hist32[b] = (int64_t)a.hist[b];
    return SW_OK;
}

// one Wolff step by "decompose everything, flip one cluster"; |C| is added to *d_size_slot (zeroed by the caller)
static int wolff_step_labelling(sw_handle* h, unsigned long long* d_size_slot, bool maintain, cudaStream_t s)
{
    const Params p = params_at(h, h->t);
    int rc = zero_sweep_counters(h, s);
    if (rc) return rc;
    rc = launch_label_front<SRC_PHILOX>(h, p, nullptr, h->d_labels, s, maintain);
    if (rc) return rc;
    if ((p.L % TW) == 0 && (p.L % TH) == 0)
        k_final<MODE_WOLFF, 0, true, true><<<dim3(p.ntx, p.nty), FIN_THREADS, 0, s>>>(p, h->d_labels, h->d_spins, h->d_acc,
                                                                                    d_size_slot, nullptr);
    else
        k_final<MODE_WOLFF, 0, false, true><<<dim3(p.ntx, p.nty), FIN_THREADS, 0, s>>>(p, h->d_labels, h->d_spins, h->d_acc,
                                                                                     d_size_slot, nullptr);
    SW_LAUNCHED(h, "k_final<WOLFF>");
    SW_PROF(h, 3, s);
    if (h->prof_on && h->prof_n < PROF_MAX) ++h->prof_n;
    ++h->t;
    return SW_OK;
}

int wolff_step(sw_handle* h, int64_t n, int64_t* h_sizes, void* stream)
{
    if (!h || n < 0) return SW_EINVAL;
    if (h->q != 2 || h->dim != 2) return SW_EINVAL;      // DESIGN.md reading 8: the paper defines Wolff for Ising only
    if (!h->bound || h->nbands > 1) return SW_ESTATE;
    DeviceGuard guard(h);
    cudaStream_t s = (cudaStream_t)stream;
    const bool front = h->wolff_levels > 0;
    int64_t done = 0;
    while (done < n) {
        const int64_t batch = (n - done) < WOLFF_RING ? (n - done) : WOLFF_RING;
        SW_CUDA(h, cudaMemsetAsync(h->d_wolff, 0, sizeof(unsigned long long) * (size_t)batch, s));
        int64_t k = 0;
        while (k < batch) {
            if (!front) {
                int rc = wolff_step_labelling(h, h->d_wolff + k, true, s);
                if (rc) return rc;
                h->last_labels = h->d_labels;
                ++k;
                continue;
            }
            // frontier growth (wolff_kernel.cuh): as many steps as finish within the level budget, in one launch
            k_wolff_front<<<1, WOLFF_THREADS, 0, s>>>(params_at(h, h->t), h->d_spins, h->d_size, h->wolff_levels,
                                                      (int)(batch - k), h->d_wolff + k, h->d_wolff_status);
            SW_LAUNCHED(h, "k_wolff_front");
            int ndone = 0;
            SW_CUDA(h, cudaMemcpyAsync(&ndone, h->d_wolff_status, sizeof(int), cudaMemcpyDeviceToHost, s));
            SW_CUDA(h, cudaStreamSynchronize(s));
            h->t += (uint64_t)ndone;
            k += ndone;
            if (k < batch) {                             // the step at counter t was given up (spins restored): label everything
                int rc = wolff_step_labelling(h, h->d_wolff + k, false, s);
                if (rc) return rc;
                ++k;
            }
            // in this mode the labels buffer and the series are not maintained (most steps label nothing)
            h->last_labels = nullptr;
            h->series_lo = h->series_hi = h->t;
        }
        if (h_sizes) {
            SW_CUDA(h, cudaMemcpyAsync(h_sizes + done, h->d_wolff, sizeof(int64_t) * (size_t)batch,
                                       cudaMemcpyDeviceToHost, s));
            SW_CUDA(h, cudaStreamSynchronize(s));
        }
        done += batch;
    }
    return SW_OK;
}

// n few-cluster steps (label_kernels.cuh: k_few_seeds + k_final<MODE_FEW>): decompose the whole lattice, select the clusters
// that hold a seed site, flip each selected cluster with probability T_flip / 2^32
int sw_fewcluster_step(sw_handle* h, int64_t n, int32_t n_seeds, uint32_t T_flip, int64_t* h_flipped, void* stream)
{
    if (!h || n < 0 || n_seeds < 0 || n_seeds > 65536) return SW_EINVAL;
    if (h->q != 2 || h->dim != 2) return SW_EINVAL;      // as wolff_step: defined for the Ising model on the square lattice
    int slots = 2;
    while (slots < 2 * n_seeds) slots *= 2;
    if ((int64_t)slots > h->N) return SW_EINVAL;         // the table of selected roots lives in the N-int cluster-size scratch
    if (!h->bound || h->nbands > 1) return SW_ESTATE;
    DeviceGuard guard(h);
    cudaStream_t s = (cudaStream_t)stream;
    int64_t done = 0;
    while (done < n) {
        const int64_t batch = (n - done) < WOLFF_RING ? (n - done) : WOLFF_RING;
        SW_CUDA(h, cudaMemsetAsync(h->d_wolff, 0, sizeof(unsigned long long) * (size_t)batch, s));
        for (int64_t k = 0; k < batch; ++k) {
            Params p = params_at(h, h->t);
            p.T_flip = T_flip; p.few_mask = slots - 1;
            int rc = zero_sweep_counters(h, s);
            if (rc) return rc;
            rc = launch_label_front<SRC_PHILOX>(h, p, nullptr, h->d_labels, s, true);
            if (rc) return rc;
            k_few_seeds<<<1, 256, 0, s>>>(p, h->d_labels, h->d_size, n_seeds);
            SW_LAUNCHED(h, "k_few_seeds");
            if ((p.L % TW) == 0 && (p.L % TH) == 0)
                k_final<MODE_FEW, 0, true, true><<<dim3(p.ntx, p.nty), FIN_THREADS, 0, s>>>(p, h->d_labels, h->d_spins, h->d_acc,
                                                                                          h->d_wolff + k, (uint32_t*)h->d_size);
            else
                k_final<MODE_FEW, 0, false, true><<<dim3(p.ntx, p.nty), FIN_THREADS, 0, s>>>(p, h->d_labels, h->d_spins, h->d_acc,
                                                                                           h->d_wolff + k, (uint32_t*)h->d_size);
            SW_LAUNCHED(h, "k_final<FEW>");
            SW_PROF(h, 3, s);
            if (h->prof_on && h->prof_n < PROF_MAX) ++h->prof_n;
            ++h->t;
            h->last_labels = h->d_labels;
        }
        if (h_flipped) {
            SW_CUDA(h, cudaMemcpyAsync(h_flipped + done, h->d_wolff, sizeof(int64_t) * (size_t)batch, cudaMemcpyDeviceToHost, s));
            SW_CUDA(h, cudaStreamSynchronize(s));
        }
        done += batch;
    }
    return SW_OK;
}

int sw_wolff_frontier(sw_handle* h, int max_levels)
{
    if (!h || max_levels < 0 || h->dim != 2) return SW_EINVAL;
    h->wolff_levels = max_levels;
    return SW_OK;
}

// The paper's own pipeline as an ablation baseline (paper_kernels.cuh): self-labelling on B x B tiles, then label relaxation
// (method 0) or hierarchical sewing (method 1), then a flatten pass.
int sw_label_paper(sw_handle* h, int method, int B, const uint8_t* d_bonds_in, int32_t* d_labels_out, sw_paper_stats* h_stats,
                   void* stream)
{
    if (!h || h->dim != 2 || (method != 0 && method != 1) || (B != 8 && B != 16 && B != 32)) return SW_EINVAL;
    if (!h->bound) return SW_ESTATE;
    const int L = h->L;
    int nt = L / B;
    if (L % B != 0 || (method == 1 && (nt & (nt - 1)) != 0)) return SW_EINVAL;       // sewing pairs tiles level by level
    DeviceGuard guard(h);
    const uint8_t* bonds = d_bonds_in ? d_bonds_in : h->d_bonds;
    int32_t* labels = d_labels_out ? d_labels_out : h->d_labels;
    if (!bonds) return SW_ESTATE;
    if (((uintptr_t)bonds | (uintptr_t)labels) & 15u) return SW_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    int* const d_flag = h->d_wolff_status + 1;           // [0] belongs to the frontier Wolff kernel; [1] changed, [2] passes
    int* const d_rlab = h->d_size;
    struct Events {                                      // destroyed on every return path
        cudaEvent_t e[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};   // [4]: before the wrap-around step of the sewing
        ~Events() { for (int k = 0; k < 5; ++k) if (e[k]) cudaEventDestroy(e[k]); }
    } evs;
    cudaEvent_t* const ev = evs.e;
    for (int k = 0; k < 5; ++k) SW_CUDA(h, cudaEventCreate(&ev[k]));
    int rc = zero_sweep_counters(h, s);
    if (rc) return rc;
    SW_CUDA(h, cudaMemsetAsync(d_flag, 0, 2 * sizeof(int), s));
    SW_CUDA(h, cudaEventRecord(ev[0], s));
    const dim3 tiles(nt, nt);
    if (B == 8)       kp_selflabel<8><<<tiles, 64, 0, s>>>(L, bonds, labels, d_rlab, d_flag + 1);
    else if (B == 16) kp_selflabel<16><<<tiles, 256, 0, s>>>(L, bonds, labels, d_rlab, d_flag + 1);
    else              kp_selflabel<32><<<tiles, 1024, 0, s>>>(L, bonds, labels, d_rlab, d_flag + 1);
    SW_LAUNCHED(h, "kp_selflabel");
    SW_CUDA(h, cudaEventRecord(ev[1], s));
    int iterations = 0, levels = 0;
    unsigned long long* const d_ncl = &h->d_acc->part[0].n_clusters;
    const int gN = grid_capped(h->N, 256, 148 * 16);
    if (method == 0) {
        const int gb = grid_capped(2 * (int64_t)nt * L, 256, 148 * 16);
        while (true) {                                   // the stopping criterion is read by the host between launches
            SW_CUDA(h, cudaMemsetAsync(d_flag, 0, sizeof(int), s));
            kp_relax<<<gb, 256, 0, s>>>(L, B, bonds, labels, d_rlab, d_flag);
            SW_LAUNCHED(h, "kp_relax");
            ++iterations;
            int changed = 0;
            SW_CUDA(h, cudaMemcpyAsync(&changed, d_flag, sizeof(int), cudaMemcpyDeviceToHost, s));
            SW_CUDA(h, cudaStreamSynchronize(s));
            if (!changed) break;
        }
        SW_CUDA(h, cudaEventRecord(ev[2], s));
        kp_flatten_relax<<<gN, 256, 0, s>>>((int)h->N, labels, d_rlab, d_ncl);
        SW_LAUNCHED(h, "kp_flatten_relax");
    } else {
        for (int Bk = B; 2 * Bk <= L; Bk *= 2) {
            kp_sew<<<dim3(L / (2 * Bk), L / (2 * Bk)), 32, 0, s>>>(L, Bk, bonds, labels);
            SW_LAUNCHED(h, "kp_sew");
            ++levels;
        }
        SW_CUDA(h, cudaEventRecord(ev[4], s));
        kp_sew_wrap<<<1, 32, 0, s>>>(L, bonds, labels);
        SW_LAUNCHED(h, "kp_sew_wrap");
        SW_CUDA(h, cudaEventRecord(ev[2], s));
        kp_flatten<<<gN, 256, 0, s>>>((int)h->N, labels, d_ncl);
        SW_LAUNCHED(h, "kp_flatten");
    }
    SW_CUDA(h, cudaEventRecord(ev[3], s));
    int passes = 0;
    SW_CUDA(h, cudaMemcpyAsync(&passes, d_flag + 1, sizeof(int), cudaMemcpyDeviceToHost, s));
    SW_CUDA(h, cudaStreamSynchronize(s));
    if (h_stats) {
        float t01 = 0.f, t12 = 0.f, t23 = 0.f;
        SW_CUDA(h, cudaEventElapsedTime(&t01, ev[0], ev[1]));
        SW_CUDA(h, cudaEventElapsedTime(&t12, ev[1], ev[2]));
        SW_CUDA(h, cudaEventElapsedTime(&t23, ev[2], ev[3]));
        h_stats->selflabel_passes_max = passes;
        h_stats->relax_iterations = iterations;
        h_stats->sewing_levels = levels;
        h_stats->ms_local = t01; h_stats->ms_consolidate = t12; h_stats->ms_flatten = t23;
        h_stats->ms_wrap = 0.0;
        if (method == 1) {
            float tw = 0.f;
            SW_CUDA(h, cudaEventElapsedTime(&tw, ev[4], ev[2]));
            h_stats->ms_wrap = tw;
        }
    }
    h->last_labels = labels;
    return SW_OK;
}

int sw_observables_ex(sw_handle* h, sw_obs* h_out, int flags, void* stream)
{
    if (!h || !h_out || (flags & ~(SW_OBS_SPINS | SW_OBS_CLUSTERS))) return SW_EINVAL;
    if (!h->bound || h->nbands > 1) return SW_ESTATE;    // (a banded handle holds its band's rows only: sw_band_counters)
    DeviceGuard guard(h);
    cudaStream_t s = (cudaStream_t)stream;
    const Params p = params_at(h, h->t);
    if (flags & SW_OBS_SPINS) {
        SW_CUDA(h, cudaMemsetAsync(&h->d_acc->sat, 0, sizeof(unsigned long long) * 9, s));
        if (h->dim == 3) k3_observables<<<grid_capped(h->N / 4, 256, 148 * 8), 256, 0, s>>>(p, h->d_spins, h->d_acc);
        else             k_observables<<<(h->L < 148 * 8 ? h->L : 148 * 8), 256, 0, s>>>(p, h->d_spins, h->d_acc);
        SW_LAUNCHED(h, "k_observables");
    }
    const bool clusters = (flags & SW_OBS_CLUSTERS) && h->last_labels;
    if (clusters) {
        int rc = cluster_stats_device(h, h->last_labels, s);
        if (rc) return rc;
    }
    Acc a;
    SW_CUDA(h, cudaMemcpyAsync(&a, h->d_acc, sizeof(Acc), cudaMemcpyDeviceToHost, s));
    SW_CUDA(h, cudaStreamSynchronize(s));
    memset(h_out, 0, sizeof(*h_out));
    const int64_t N = h->N;
    if (flags & SW_OBS_SPINS) {
        h_out->sat_bonds = (int64_t)a.sat;
        int64_t rest = 0;
        for (int k = 1; k < h->q; ++k) { h_out->state_count[k] = (int64_t)a.cnt[k]; rest += (int64_t)a.cnt[k]; }
        h_out->state_count[0] = N - rest;
        if (h->q == 2) {
            h_out->energy = -(2 * h_out->sat_bonds - (int64_t)h->dim * N);
            h_out->magnetisation = h_out->state_count[0] - h_out->state_count[1];
        } else {
            int64_t mx = 0;
            for (int k = 0; k < h->q; ++k) if (h_out->state_count[k] > mx) mx = h_out->state_count[k];
            h_out->energy = -h_out->sat_bonds;
            h_out->magnetisation = (int64_t)h->q * mx - N;
        }
    }
    if (h->last_labels) {                                // counted by the labelling itself: free
        for (int k = 0; k < ACC_PARTS; ++k) {
            h_out->n_clusters += (int64_t)a.part[k].n_clusters;
            h_out->n_active_bonds += (int64_t)a.part[k].n_active;
        }
    }
    if (clusters) {
        h_out->max_cluster = (int64_t)a.cs_max;
        h_out->sum_sq_cluster = a.cs_sumsq;
    }
    h_out->counter = h->t;
    return SW_OK;
}

int sw_observables(sw_handle* h, sw_obs* h_out, void* stream)
{
    return sw_observables_ex(h, h_out, SW_OBS_SPINS | SW_OBS_CLUSTERS, stream);
}

int sw_series_read(sw_handle* h, uint64_t t_first, int64_t n, int64_t* h_energy, int64_t* h_magnetisation, void* stream)
{
    if (!h || n < 0 || (n > 0 && !h_energy) || (h->q != 2 && h_magnetisation)) return SW_EINVAL;
    if (!h->bound) return SW_ESTATE;
    DeviceGuard guard(h);
    if (n == 0) return SW_OK;
    if (t_first < h->series_lo || t_first + (uint64_t)n > h->series_hi) return SW_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    SeriesEntry* buf = new (std::nothrow) SeriesEntry[(size_t)n];
    if (!buf) return SW_ENOMEM;
    const uint64_t i0 = t_first & (SERIES_RING - 1);
    const uint64_t n1 = (uint64_t)n < SERIES_RING - i0 ? (uint64_t)n : SERIES_RING - i0;      // up to the end of the ring
    cudaError_t e = cudaMemcpyAsync(buf, h->d_series + i0, sizeof(SeriesEntry) * n1, cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess && n1 < (uint64_t)n)
        e = cudaMemcpyAsync(buf + n1, h->d_series, sizeof(SeriesEntry) * ((uint64_t)n - n1), cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) { delete[] buf; return cuda_fail(h, e, "sw_series_read"); }
    const int64_t N = h->N;
    for (int64_t k = 0; k < n; ++k) {
        const int64_t sat = (int64_t)buf[k].sat;
        h_energy[k] = h->q == 2 ? -(2 * sat - (int64_t)h->dim * N) : -sat;
        if (h_magnetisation) h_magnetisation[k] = N - 2 * (int64_t)buf[k].minus;
    }
    delete[] buf;
    return SW_OK;
}

int sw_sweep_host(sw_handle* h, const void* h_spins_in, int64_t n, void* h_spins_out, int32_t* h_labels_out,
                  sw_obs* h_obs, void* stream)
{
    return sw_sweep_host_ex(h, h_spins_in, n, h_spins_out, h_labels_out, h_obs, SW_OBS_SPINS | SW_OBS_CLUSTERS, stream);
}

int sw_sweep_host_ex(sw_handle* h, const void* h_spins_in, int64_t n, void* h_spins_out, int32_t* h_labels_out,
                     sw_obs* h_obs, int obs_flags, void* stream)
{
    if (!h || n < 0) return SW_EINVAL;
    if (!h->bound) return SW_ESTATE;
    DeviceGuard guard(h);
    cudaStream_t s = (cudaStream_t)stream;
    if (h_spins_in) SW_CUDA(h, cudaMemcpyAsync(h->d_spins, h_spins_in, (size_t)h->N, cudaMemcpyHostToDevice, s));
    int rc = sw_sweep(h, n, stream);
    if (rc) return rc;
    if (h_spins_out) SW_CUDA(h, cudaMemcpyAsync(h_spins_out, h->d_spins, (size_t)h->N, cudaMemcpyDeviceToHost, s));
    if (h_labels_out)
        SW_CUDA(h, cudaMemcpyAsync(h_labels_out, h->d_labels, (size_t)h->N * sizeof(int32_t), cudaMemcpyDeviceToHost, s));
    if (h_obs) return sw_observables_ex(h, h_obs, obs_flags, stream);
    SW_CUDA(h, cudaStreamSynchronize(s));
    return SW_OK;
}

}  // extern "C"

// ---- sw_cluster_stats_static: cluster statistics with the scratch compiled into the library (include/swb200.h) -----------
// For callers that cannot allocate device memory (see the header).  Everything the two cluster kernels need beyond the labels
// and the result -- the accumulators and one int32 per site -- lives in the array below.  Its name is only a handle on the
// host side: the kernels get the device address that cudaGetSymbolAddress returns for the GPU that is current, looked up once
// per GPU.  Nothing here calls cudaMalloc, cudaFree or an allocating routine.
namespace {

constexpr int STATIC_ACC_INTS = (int)((sizeof(Acc) + 255) / 256 * 256 / sizeof(int));   // the Acc, padded to 256 bytes
static_assert(STATIC_ACC_INTS * sizeof(int) >= sizeof(Acc), "the accumulators fit in front of the size array");
static __device__ __align__(256) int g_static_scratch[STATIC_ACC_INTS + SW_STATIC_MAX_SITES];

constexpr int STATIC_MAX_DEVICES = 64;
std::mutex g_static_mutex;                                // guards the table below (first calls from several host threads)
int* g_static_ptr[STATIC_MAX_DEVICES];                    // device address of g_static_scratch on GPU d; NULL: not looked up yet

// accumulators of k_cluster_stats -> the caller's sw_cstats (one warp; bin b by lane b)
__global__ void k_cstats_emit(const Acc* __restrict__ acc, sw_cstats* __restrict__ out)
{
    out->hist32[threadIdx.x] = (int64_t)acc->hist[threadIdx.x];
    if (threadIdx.x == 0) {
        out->n_clusters = (int64_t)acc->cs_nclusters;
        out->max_cluster = (int64_t)acc->cs_max;
        out->sum_sq_cluster = acc->cs_sumsq;
    }
}

}  // namespace

extern "C" int sw_cluster_stats_static(int32_t L, const int32_t* d_labels, sw_cstats* d_out, void* stream)
{
    if (L < 4 || (L % 4) != 0 || !d_labels || !d_out) return SW_EINVAL;
    if (((uintptr_t)d_labels & 15u) || ((uintptr_t)d_out & 7u)) return SW_EINVAL;
    const int64_t N = (int64_t)L * L;
    if (N > (int64_t)SW_STATIC_MAX_SITES) return SW_ELIMIT;
    cudaPointerAttributes at_in, at_out;
    if (cudaPointerGetAttributes(&at_in, d_labels) != cudaSuccess || cudaPointerGetAttributes(&at_out, d_out) != cudaSuccess) {
        cudaGetLastError();
        return SW_EINVAL;
    }
    const bool dev_in = at_in.type == cudaMemoryTypeDevice || at_in.type == cudaMemoryTypeManaged;
    const bool dev_out = at_out.type == cudaMemoryTypeDevice || at_out.type == cudaMemoryTypeManaged;
    if (!dev_in || !dev_out || at_in.device != at_out.device) return SW_EINVAL;
    const int dev = at_in.device;
    if (dev < 0 || dev >= STATIC_MAX_DEVICES) return SW_EINVAL;
    // make the GPU of the buffers current for the call (as every handle entry point does), restore the caller's afterwards
    struct Current {
        int prev = -1; bool switched = false;
        ~Current() { if (switched) cudaSetDevice(prev); }
    } cur;
    if (cudaGetDevice(&cur.prev) != cudaSuccess) return SW_ECUDA;
    if (cur.prev != dev) {
        if (cudaSetDevice(dev) != cudaSuccess) return SW_ECUDA;
        cur.switched = true;
    }
    int* scratch = nullptr;
    {   // set-up, once per GPU, with that GPU current: the device address of the array (its host-side name is not one)
        std::lock_guard<std::mutex> lock(g_static_mutex);
        if (!g_static_ptr[dev]) {
            void* ptr = nullptr;
            if (cudaGetSymbolAddress(&ptr, g_static_scratch) != cudaSuccess || !ptr) {
                cudaGetLastError();
                return SW_ECUDA;
            }
            g_static_ptr[dev] = (int*)ptr;
        }
        scratch = g_static_ptr[dev];
    }
    Acc* const acc = reinterpret_cast<Acc*>(scratch);
    int* const size = scratch + STATIC_ACC_INTS;
    cudaStream_t s = (cudaStream_t)stream;
    Params p;
    memset(&p, 0, sizeof(p));
    p.L = L; p.N = (int32_t)N; p.H = L; p.q = 2; p.logL = -1;
    p.ntx = (L + TW - 1) / TW; p.nty = (L + TH - 1) / TH; p.nband = p.nty;
    // the array still holds the previous call's sizes and sums: clear the accumulators and the N entries used now
    if (cudaMemsetAsync(scratch, 0, ((size_t)STATIC_ACC_INTS + (size_t)N) * sizeof(int), s) != cudaSuccess) return SW_ECUDA;
    k_cluster_sizes<<<dim3(p.ntx, p.nty), 256, 0, s>>>(p, d_labels, size);
    if (cudaGetLastError() != cudaSuccess) return SW_ECUDA;
    k_cluster_stats<<<grid_capped(N, 256, 148 * 8), 256, 0, s>>>(p, d_labels, size, acc);
    if (cudaGetLastError() != cudaSuccess) return SW_ECUDA;
    k_cstats_emit<<<1, 32, 0, s>>>(acc, d_out);
    if (cudaGetLastError() != cudaSuccess) return SW_ECUDA;
    return SW_OK;
}
